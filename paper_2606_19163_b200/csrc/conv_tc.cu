// conv_tc.cu - tcgen05 / TMEM / TMA implicit-GEMM convolution for sm_100a (bf16 in, fp32
// accumulate).  One kernel serves 3x3 / 1x1 fprop on a single or dual source (the channel
// concat with the cached skip is fused into the operand loader: K blocks below c0 come from
// h's tensor map, the rest from the skip's - PAPER.md:L91, north_star), stride-1 dgrad (fprop
// with flipped/transposed weights), stride-2 fprop (5-D parity view of the input) and
// stride-2 dgrad (4 output-parity phases, each a sub-pixel conv with 1/2/2/4 taps).
//
// GEMM view: D[pixel, co] = sum_{tap, c} A[pixel shifted by tap, c] * W[co][tap][c]
//   M tile = 128 output pixels = a (bn x bh x bw) box of the NHWC tensor, loaded per tap by
//            ONE tiled TMA with shifted coordinates; out-of-bounds rows/cols are zero-filled
//            by TMA, which implements pad = 1 for free,
//   N tile = BN output channels (160: every channel count of the configs is 320 k),
//   K block = 64 channels of one tap (128-byte swizzled rows, K-major for both operands).
// Warp roles (192 threads): warp 0 TMA producer, warp 1 MMA issuer (one elected thread;
// owns TMEM alloc), warps 2-5 epilogue (tcgen05.ld -> +bias +temb/residual -> bf16 ->
// global).  Persistent over tiles with two TMEM accumulators so the epilogue of tile i
// overlaps the main loop of tile i+1.
#include <cuda.h>

#include <map>
#include <mutex>
#include <string>
#include <vector>

#include "common.cuh"
#include "kernels.h"
#include "sm100.cuh"
#include "tmap.h"

namespace pulse {

namespace {

using namespace sm100;
using namespace tmap;

constexpr int BM = 128, BK = 64;
constexpr int A_BYTES = BM * BK * 2;           // 16 KB

struct TcParams {      // phases: see conv_tc2.cu
  int c0_blocks, c_blocks, ctot, c0;
  int s2;                         // 1: stride-2 fprop through the 5-D parity view
  int nph, ph_tap0[5], ph_wrow[4], ph_ooy[4], ph_oox[4];
  Tap taps[16];
  int bw, bh, bn, tiles_h, tiles_mn, n_tiles;
  int GH, GN;                     // pixel grid (rows, images); columns == bw
  const bf16* bias; const float* pn; const bf16* residual; bf16* out; int accumulate;
  int OH, OW, osy, osx, cout_total;
};

template <int BN> struct Cfg {
  static constexpr int B_BYTES = BN * BK * 2;
  static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
  static constexpr int STAGES = (220 * 1024) / STAGE_BYTES > 8 ? 8 : (220 * 1024) / STAGE_BYTES;
  static constexpr int SMEM = STAGES * STAGE_BYTES + 1024;
  static constexpr int TMEM_COLS = 2 * BN <= 256 ? 256 : 512;
};

template <int BN>
__global__ void __launch_bounds__(192, 1)
conv_tc_k(const __grid_constant__ CUtensorMap mapA0, const __grid_constant__ CUtensorMap mapA1,
          const __grid_constant__ CUtensorMap mapB, const TcParams p) {
  using C = Cfg<BN>;
  extern __shared__ uint8_t smem_raw[];
  __shared__ uint64_t full_bar[C::STAGES], empty_bar[C::STAGES], tfull_bar[2], tempty_bar[2];
  __shared__ uint32_t tmem_base_s;
  uint8_t* smem = smem_raw + ((1024 - (smem_u32(smem_raw) & 1023)) & 1023);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int tiles_ph = p.tiles_mn * p.n_tiles;      // tiles per phase
  const int total_tiles = p.nph * tiles_ph;

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&mapA0); prefetch_tmap(&mapA1); prefetch_tmap(&mapB);
    for (int i = 0; i < C::STAGES; ++i) { mbar_init(&full_bar[i], 1); mbar_init(&empty_bar[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&tfull_bar[i], 1); mbar_init(&tempty_bar[i], 4); }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc(&tmem_base_s, C::TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_s;
  pdl_wait();                  // everything above overlapped the tail of the previous kernel
  pdl_launch_dependents();

  if (warp == 0) {
    if (lane == 0) {
      // ===== TMA producer =====
      int stage = 0; uint32_t phase = 0;
      for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
        const int ph = tile / tiles_ph, tl = tile - ph * tiles_ph;
        const int mt = tl / p.n_tiles, nt = tl - mt * p.n_tiles;
        const int n0 = (mt / p.tiles_h) * p.bn, y0 = (mt % p.tiles_h) * p.bh;
        const int tap0 = p.ph_tap0[ph], num_kb = (p.ph_tap0[ph + 1] - tap0) * p.c_blocks, wrow = p.ph_wrow[ph];
        for (int kb = 0; kb < num_kb; ++kb) {
          const int ti = kb / p.c_blocks, cb = kb - ti * p.c_blocks;
          const Tap t = p.taps[tap0 + ti];
          mbar_wait(&empty_bar[stage], phase ^ 1);
          mbar_expect_tx(&full_bar[stage], C::STAGE_BYTES);
          uint8_t* sa = smem + stage * C::STAGE_BYTES;
          const bool first = cb < p.c0_blocks;
          const CUtensorMap* ma = first ? &mapA0 : &mapA1;
          const int cch = (first ? cb : cb - p.c0_blocks) * BK;
          if (!p.s2) tma_load_4d(sa, ma, &full_bar[stage], cch, t.dx, y0 + t.dy, n0);
          else tma_load_5d(sa, ma, &full_bar[stage], t.px * p.c0 + cch, t.dx, t.py, y0 + t.dy, n0);
          tma_load_2d(sa + A_BYTES, &mapB, &full_bar[stage], t.widx * p.ctot + cb * BK, wrow + nt * BN);
          if (++stage == C::STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    {
      // ===== MMA issuer: the whole warp runs the loop, one elected lane issues (sm100.cuh elect_one_sync) =====
      constexpr uint32_t idesc = idesc_bf16(BM, BN, 0, 0);
      constexpr uint64_t dbase = smem_desc_sw128(16, 1024);
      int stage = 0; uint32_t phase = 0; int acc = 0; uint32_t acc_phase = 0;
      for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
        const int ph = tile / tiles_ph;
        const int num_kb = (p.ph_tap0[ph + 1] - p.ph_tap0[ph]) * p.c_blocks;
        mbar_wait(&tempty_bar[acc], acc_phase ^ 1);
        tc_fence_after();
        const uint32_t tmem_d = tmem_base + acc * BN;
        for (int kb = 0; kb < num_kb; ++kb) {
          mbar_wait(&full_bar[stage], phase);
          tc_fence_after();
          const uint32_t a_addr = smem_u32(smem + stage * C::STAGE_BYTES), b_addr = a_addr + A_BYTES;
          if (elect_one_sync()) {
#pragma unroll
            for (int k = 0; k < BK / 16; ++k)
              umma_bf16(tmem_d, desc_with_addr(dbase, a_addr + k * 32), desc_with_addr(dbase, b_addr + k * 32), idesc,
                        (kb | k) != 0);
            umma_commit(&empty_bar[stage]);
            if (kb == num_kb - 1) umma_commit(&tfull_bar[acc]);
          }
          __syncwarp();
          if (++stage == C::STAGES) { stage = 0; phase ^= 1; }
        }
        acc ^= 1;
        if (acc == 0) acc_phase ^= 1;
      }
    }
  } else {
    // ===== epilogue: warps 2..5 own TMEM lane quadrants (warp % 4) =====
    const int q = warp & 3;
    const int row = q * 32 + lane;
    const int n_l = row / (p.bh * p.bw), rem = row - n_l * (p.bh * p.bw);
    const int y_l = rem / p.bw, x = rem - y_l * p.bw;
    int acc = 0; uint32_t acc_phase = 0;
    for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
      const int ph = tile / tiles_ph, tl = tile - ph * tiles_ph;
      const int mt = tl / p.n_tiles, nt = tl - mt * p.n_tiles;
      const int n = (mt / p.tiles_h) * p.bn + n_l, y = (mt % p.tiles_h) * p.bh + y_l;
      const bool valid = n < p.GN && y < p.GH;
      const size_t off = (((size_t)n * p.OH + (size_t)y * p.osy + p.ph_ooy[ph]) * p.OW + (size_t)x * p.osx + p.ph_oox[ph]) *
                             p.cout_total + (size_t)nt * BN;
      mbar_wait(&tfull_bar[acc], acc_phase);
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + acc * BN;
#pragma unroll 1
      for (int ch = 0; ch < BN / 32; ++ch) {
        uint32_t r[32];
        tmem_ld32(taddr + ch * 32, r);
        tmem_ld_wait();
        if (ch == BN / 32 - 1) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(&tempty_bar[acc]);
        }
        if (valid) {
          const int co = nt * BN + ch * 32;
          float v[32];
#pragma unroll
          for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
          if (p.bias) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              float b[8];
              ldv(p.bias + co + i * 8, b);
#pragma unroll
              for (int j = 0; j < 8; ++j) v[i * 8 + j] += b[j];
            }
          }
          if (p.pn) {
            const float4* pp = reinterpret_cast<const float4*>(p.pn + (size_t)n * p.cout_total + co);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              const float4 t = pp[i];
              v[i * 4] += t.x; v[i * 4 + 1] += t.y; v[i * 4 + 2] += t.z; v[i * 4 + 3] += t.w;
            }
          }
          if (p.residual) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              float b[8];
              ldv(p.residual + off + ch * 32 + i * 8, b);
#pragma unroll
              for (int j = 0; j < 8; ++j) v[i * 8 + j] += b[j];
            }
          }
          if (p.accumulate) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              float b[8];
              ldv(p.out + off + ch * 32 + i * 8, b);
#pragma unroll
              for (int j = 0; j < 8; ++j) v[i * 8 + j] += b[j];
            }
          }
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            float o[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) o[j] = v[i * 8 + j];
            stv(p.out + off + ch * 32 + i * 8, o);
          }
        }
      }
      acc ^= 1;
      if (acc == 0) acc_phase ^= 1;
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, C::TMEM_COLS);
  }
}

}  // namespace

// ------------------------------------------------------------------------------ host: tensor maps
namespace tmap {
namespace {
typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                             const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                             CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
std::string g_tc_err;
EncodeFn g_encode = nullptr;
std::mutex g_mu;
std::map<std::vector<uint64_t>, CUtensorMap> g_maps;
int g_sms = 0;

bool init_driver() {
  if (g_encode) return true;
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) {
    g_tc_err = "cuTensorMapEncodeTiled not available";
    return false;
  }
  g_encode = (EncodeFn)fn;
  return true;
}
}  // namespace

void set_error(const std::string& e) { g_tc_err = e; }
int sm_count() {
  if (!g_sms) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&g_sms, cudaDevAttrMultiProcessorCount, dev);
    if (g_sms <= 0) g_sms = 148;
  }
  return g_sms;
}

bool get_map(const void* ptr, int rank, const uint64_t* dims, const uint64_t* strides, const uint32_t* box,
             CUtensorMap* out, int swizzle_bytes, int elem_bytes) {
  std::vector<uint64_t> key;
  key.push_back((uint64_t)ptr); key.push_back(rank + 16 * (uint64_t)swizzle_bytes + 4096 * (uint64_t)elem_bytes);
  for (int i = 0; i < rank; ++i) { key.push_back(dims[i]); key.push_back(box[i]); if (i) key.push_back(strides[i - 1]); }
  std::lock_guard<std::mutex> lk(g_mu);
  auto it = g_maps.find(key);
  if (it != g_maps.end()) { *out = it->second; return true; }
  if (!init_driver()) return false;
  cuuint64_t gd[5], gs[4]; cuuint32_t bx[5], es[5];
  for (int i = 0; i < rank; ++i) { gd[i] = dims[i]; bx[i] = box[i]; es[i] = 1; if (i) gs[i - 1] = strides[i - 1]; }
  CUtensorMap m;
  CUresult r = g_encode(&m, elem_bytes == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, rank, const_cast<void*>(ptr), gd, gs, bx, es,
                        CU_TENSOR_MAP_INTERLEAVE_NONE,
                        swizzle_bytes == 128 ? CU_TENSOR_MAP_SWIZZLE_128B
                                             : (swizzle_bytes == 64 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_NONE),
                        CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    g_tc_err = "cuTensorMapEncodeTiled failed with " + std::to_string((int)r);
    return false;
  }
  if (g_maps.size() > 4096) g_maps.clear();
  g_maps[key] = m;
  *out = m;
  return true;
}

bool act_map(const void* ptr, int n, int h, int w, int c, int bw, int bh, int bn, CUtensorMap* out) {
  uint64_t dims[4] = {(uint64_t)c, (uint64_t)w, (uint64_t)h, (uint64_t)n};
  uint64_t str[3] = {(uint64_t)c * 2, (uint64_t)w * c * 2, (uint64_t)h * w * c * 2};
  uint32_t box[4] = {64, (uint32_t)bw, (uint32_t)bh, (uint32_t)bn};
  return get_map(ptr, 4, dims, str, box, out);
}
bool act_map_s2(const void* ptr, int n, int h, int w, int c, int bw, int bh, int bn, CUtensorMap* out) {
  uint64_t dims[5] = {(uint64_t)2 * c, (uint64_t)w / 2, 2, (uint64_t)h / 2, (uint64_t)n};
  uint64_t str[4] = {(uint64_t)2 * c * 2, (uint64_t)w * c * 2, (uint64_t)2 * w * c * 2, (uint64_t)h * w * c * 2};
  uint32_t box[5] = {64, (uint32_t)bw, 1, (uint32_t)bh, (uint32_t)bn};
  return get_map(ptr, 5, dims, str, box, out);
}
bool mat_map(const void* ptr, uint64_t rows, uint64_t k, int brows, CUtensorMap* out) {
  uint64_t dims[2] = {k, rows};
  uint64_t str[1] = {k * 2};
  uint32_t box[2] = {64, (uint32_t)brows};
  return get_map(ptr, 2, dims, str, box, out);
}
bool mat_map_f32(const void* ptr, uint64_t rows, uint64_t cols, int bcols, int brows, CUtensorMap* out) {
  uint64_t dims[2] = {cols, rows};
  uint64_t str[1] = {cols * 4};
  uint32_t box[2] = {(uint32_t)bcols, (uint32_t)brows};
  return get_map(ptr, 2, dims, str, box, out, 0, 4);
}
bool tile_geometry(int gh, int gw, int& bw, int& bh, int& bn) {
  if (gw < 8 || gw > 128 || (gw & (gw - 1))) return false;
  bw = gw;
  const int rows = 128 / gw;
  if (rows <= gh) { bh = rows; bn = 1; return true; }
  if ((gh & (gh - 1)) || 128 % (gh * gw)) return false;
  bh = gh; bn = 128 / (gh * gw);
  return true;
}
const std::string& last_error() { return g_tc_err; }
// 64-pixel tiles of an [n, gh, gw] grid (wgrad K blocks)
bool tile_geometry64(int gh, int gw, int& bw, int& bh, int& bn) {
  if (gw < 8 || (gw & (gw - 1))) return false;
  if (gw >= 64) { bw = 64; bh = 1; bn = 1; return gw % 64 == 0 && gw <= 256; }
  bw = gw;
  const int rows = 64 / gw;
  if (rows <= gh) { bh = rows; bn = 1; return true; }
  if ((gh & (gh - 1)) || 64 % (gh * gw)) return false;
  bh = gh; bn = 64 / (gh * gw);
  return true;
}
// NHWC activation as (c, w, h, n) with a (cbox, bw, bh, bn) box; swizzle = 2 * cbox bytes
bool act_map_c(const void* ptr, int n, int h, int w, int c, int cbox, int bw, int bh, int bn, CUtensorMap* out) {
  uint64_t dims[4] = {(uint64_t)c, (uint64_t)w, (uint64_t)h, (uint64_t)n};
  uint64_t str[3] = {(uint64_t)c * 2, (uint64_t)w * c * 2, (uint64_t)h * w * c * 2};
  uint32_t box[4] = {(uint32_t)cbox, (uint32_t)bw, (uint32_t)bh, (uint32_t)bn};
  return get_map(ptr, 4, dims, str, box, out, 2 * cbox);
}
bool act_map_s2_c(const void* ptr, int n, int h, int w, int c, int cbox, int bw, int bh, int bn, CUtensorMap* out) {
  uint64_t dims[5] = {(uint64_t)2 * c, (uint64_t)w / 2, 2, (uint64_t)h / 2, (uint64_t)n};
  uint64_t str[4] = {(uint64_t)2 * c * 2, (uint64_t)w * c * 2, (uint64_t)2 * w * c * 2, (uint64_t)h * w * c * 2};
  uint32_t box[5] = {(uint32_t)cbox, (uint32_t)bw, 1, (uint32_t)bh, (uint32_t)bn};
  return get_map(ptr, 5, dims, str, box, out, 2 * cbox);
}
}  // namespace tmap

namespace {
int pick_bn(int cout) { return cout % 160 == 0 ? 160 : (cout % 128 == 0 ? 128 : 0); }

template <int BN>
bool launch(const CUtensorMap& a0, const CUtensorMap& a1, const CUtensorMap& b, const TcParams& p, cudaStream_t st) {
  static bool attr_set = false;
  if (!attr_set) {
    if (cudaFuncSetAttribute(conv_tc_k<BN>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg<BN>::SMEM) != cudaSuccess) {
      tmap::set_error("cudaFuncSetAttribute(max dynamic smem) failed");
      return false;
    }
    attr_set = true;
  }
  const int tiles = p.nph * p.tiles_mn * p.n_tiles;
  const int grid = tiles < sm_count() ? tiles : sm_count();
  launch_pdl(conv_tc_k<BN>, dim3(grid), dim3(192), Cfg<BN>::SMEM, st, a0, a1, b, p);
  return true;
}

}  // namespace

const char* tc_last_error() { return tmap::last_error().c_str(); }

bool conv_tc_supported(const ConvArgs& a) {
  if (a.dt != DT_BF16) return false;
  if (a.src.c0 % 64 || a.src.c1 % 64 || a.src.c0 == 0) return false;
  if (!pick_bn(a.cout)) return false;
  if (a.ksize != 1 && a.ksize != 3) return false;
  int bw, bh, bn;
  if (a.mode == CONV_UP2_DGRAD) {
    if (a.ksize != 3 || a.src.c1 || (a.hin & 1) || (a.win & 1) || a.hout * 2 != a.hin || a.wout * 2 != a.win) return false;
    return tile_geometry(a.hout, a.wout, bw, bh, bn);
  }
  if (a.mode == CONV_DGRAD_S2 || a.mode == CONV_UP2) {
    if (a.ksize != 3 || a.src.c1) return false;
    if (a.hout != 2 * a.hin || a.wout != 2 * a.win) return false;
    return tile_geometry(a.hin, a.win, bw, bh, bn);
  }
  if (a.stride == 2) {
    if (a.ksize != 3 || a.src.c1 || (a.hin & 1) || (a.win & 1) || a.hout * 2 != a.hin || a.wout * 2 != a.win) return false;
  } else if (a.stride != 1 || a.hout != a.hin || a.wout != a.win) {
    return false;
  }
  return tile_geometry(a.hout, a.wout, bw, bh, bn);
}

int conv_tc(const ConvArgs& a, cudaStream_t st) {
  TcParams p;
  memset(&p, 0, sizeof p);
  const int bnn = pick_bn(a.cout);
  const bool s2d = a.mode == CONV_DGRAD_S2, up2 = a.mode == CONV_UP2, up2d = a.mode == CONV_UP2_DGRAD;
  const bool s2f = up2d || (a.mode == CONV_FPROP && a.stride == 2);      // source read through the 5-D parity view
  const int gh = (s2d || up2) ? a.hin : a.hout, gw = (s2d || up2) ? a.win : a.wout;
  tile_geometry(gh, gw, p.bw, p.bh, p.bn);
  p.c0 = a.src.c0; p.ctot = a.src.c(); p.c0_blocks = a.src.c0 / 64; p.c_blocks = p.ctot / 64;
  p.s2 = s2f;
  p.tiles_h = (gh + p.bh - 1) / p.bh;
  p.tiles_mn = p.tiles_h * ((a.n + p.bn - 1) / p.bn);
  p.n_tiles = a.cout / bnn;
  p.GH = gh; p.GN = a.n;
  p.bias = (const bf16*)a.bias; p.pn = a.pn; p.residual = (const bf16*)a.residual; p.out = (bf16*)a.out;
  p.accumulate = a.accumulate;
  CUtensorMap m0, m1, mb;
  bool ok = true;
  if (s2f) ok = act_map_s2(a.src.p0, a.n, a.hin, a.win, a.src.c0, p.bw, p.bh, p.bn, &m0);
  else ok = act_map(a.src.p0, a.n, a.hin, a.win, a.src.c0, p.bw, p.bh, p.bn, &m0);
  m1 = m0;
  if (ok && a.src.c1) ok = act_map(a.src.p1, a.n, a.hin, a.win, a.src.c1, p.bw, p.bh, p.bn, &m1);
  const uint64_t wk = (uint64_t)(up2 ? 4 : up2d ? 16 : a.ksize * a.ksize) * p.ctot;     // K of the weight matrix
  if (ok) ok = mat_map(a.w, (uint64_t)(up2 ? 4 : 1) * a.cout, wk, bnn, &mb);
  if (!ok) return -1;
  // phases (see conv_tc2.cu): taps, weight rows and output parity of each sub-pixel conv of this launch
  p.OH = a.hout; p.OW = a.wout; p.osy = p.osx = 1; p.cout_total = a.cout;
  p.nph = 0; p.ph_tap0[0] = 0;
  int ntaps = 0;
  auto add_tap = [&](int dy, int dx, int py, int px, int widx) {
    Tap t; t.dy = dy; t.dx = dx; t.py = py; t.px = px; t.widx = widx;
    p.taps[ntaps++] = t;
  };
  auto end_phase = [&](int wrow, int ooy, int oox) {
    p.ph_wrow[p.nph] = wrow; p.ph_ooy[p.nph] = ooy; p.ph_oox[p.nph] = oox;
    p.ph_tap0[++p.nph] = ntaps;
  };
  if (up2) {
    p.osy = p.osx = 2;
    for (int ph = 0; ph < 4; ++ph) {
      const int py = ph >> 1, px = ph & 1;
      for (int t = 0; t < 4; ++t) add_tap((t >> 1) - 1 + py, (t & 1) - 1 + px, 0, 0, t);
      end_phase(ph * a.cout, py, px);
    }
  } else if (up2d) {
    for (int q = 0; q < 16; ++q) {
      const int py = q >> 3, px = (q >> 2) & 1, ta = (q >> 1) & 1, tb = q & 1;
      add_tap(1 - ta - py, 1 - tb - px, py, px, q);
    }
    end_phase(0, 0, 0);
  } else if (s2d) {
    p.osy = p.osx = 2;
    const int order[4][2] = {{1, 1}, {1, 0}, {0, 1}, {0, 0}};
    for (int o = 0; o < 4; ++o) {
      const int py = order[o][0], px = order[o][1];
      for (int r = 0; r < 3; ++r) {
        if ((py + r - 1) & 1) continue;
        for (int s_ = 0; s_ < 3; ++s_) {
          if ((px + s_ - 1) & 1) continue;
          add_tap((py + r - 1) >> 1, (px + s_ - 1) >> 1, 0, 0, r * 3 + s_);
        }
      }
      end_phase(0, py, px);
    }
  } else {
    const int pad = (a.ksize - 1) / 2;
    for (int r = 0; r < a.ksize; ++r)
      for (int s_ = 0; s_ < a.ksize; ++s_) {
        if (!s2f) add_tap(r - pad, s_ - pad, 0, 0, r * a.ksize + s_);
        else add_tap(r == 0 ? -1 : 0, s_ == 0 ? -1 : 0, r == 1 ? 0 : 1, s_ == 1 ? 0 : 1, r * a.ksize + s_);
      }
    end_phase(0, 0, 0);
  }
  const bool r = bnn == 160 ? launch<160>(m0, m1, mb, p, st) : launch<128>(m0, m1, mb, p, st);
  return r ? 1 : -1;
}

// ================================================================================ wgrad
// dW[co][tap][c] += sum_pixels g[pixel, co] * in[pixel shifted by tap, c]
// GEMM view: D[128 rows = 2 x (tap, 64-channel block)][320 cols = co] += A^T B over K = pixels.
// Both operands have the channel dimension contiguous, i.e. they are MN-major: the same TMA
// boxes as fprop ([64 pixels][64 channels], 128-byte swizzled rows) are consumed directly with
// MN-major UMMA descriptors (LBO = stride between 64-channel blocks, SBO = 8 pixel rows).
// Split-K over pixel tiles fills the machine; partial tiles are reduced with fp32 red.global.add
// into dW, which is also how weight gradients accumulate across microbatches (row a11).
namespace {

constexpr int WG_PIX = 64;                 // K per stage
constexpr int WG_BLK = WG_PIX * 128;       // one [64 px][64 ch] box = 8 KB
constexpr int WG_N = 320;
constexpr int WG_STAGE = 2 * WG_BLK + (WG_N / 64) * WG_BLK;    // 56 KB
constexpr int WG_STAGES = 4;
constexpr int WG_SMEM = WG_STAGES * WG_STAGE + 1024;

struct WgParams {
  int units, c_blocks, c0_blocks, c0, ctot, ktot, s2;
  Tap taps[9];
  int bw, bh, bn, tiles_w, tiles_h;
  int pix_tiles, m_tiles, n_tiles;
  long long work;          // m_tiles * n_tiles * pix_tiles work items of (128 rows x 320 cols x 64 pixels)
  float* dw;
};

// Work distribution ("stream-K"): the work items, ordered (output tile, pixel tile), are cut into gridDim.x equal
// contiguous ranges, so every SM gets the same number of MMAs whatever the number of output tiles is (23 or 45 for
// the config-2 shapes: any whole-tile split leaves a ragged second wave).  A range that crosses an output-tile
// boundary flushes its accumulator (fp32 red.add into dW) and starts the next tile.
__global__ void __launch_bounds__(192, 1)
wgrad_tc_k(const __grid_constant__ CUtensorMap mapA0, const __grid_constant__ CUtensorMap mapA1,
           const __grid_constant__ CUtensorMap mapG, const WgParams p) {
  extern __shared__ uint8_t smem_raw[];
  __shared__ uint64_t full_bar[WG_STAGES], empty_bar[WG_STAGES], tfull_bar, tempty_bar;
  __shared__ uint32_t tmem_base_s;
  uint8_t* smem = smem_raw + ((1024 - (smem_u32(smem_raw) & 1023)) & 1023);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long wb = p.work * blockIdx.x / gridDim.x, we = p.work * (blockIdx.x + 1) / gridDim.x;

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&mapA0); prefetch_tmap(&mapA1); prefetch_tmap(&mapG);
    for (int i = 0; i < WG_STAGES; ++i) { mbar_init(&full_bar[i], 1); mbar_init(&empty_bar[i], 1); }
    mbar_init(&tfull_bar, 1); mbar_init(&tempty_bar, 4);
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc(&tmem_base_s, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_s;

  if (warp == 0) {
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0;
      for (long long w = wb; w < we; ++w) {
        const int ot = (int)(w / p.pix_tiles), pt = (int)(w - (long long)ot * p.pix_tiles);
        const int nt = ot % p.n_tiles, mt = ot / p.n_tiles;
        const int u0 = 2 * mt, u1 = min(u0 + 1, p.units - 1);
        const int tx = pt % p.tiles_w, ty = (pt / p.tiles_w) % p.tiles_h, tn = pt / (p.tiles_w * p.tiles_h);
        const int x0 = tx * p.bw, y0 = ty * p.bh, n0 = tn * p.bn;
        mbar_wait(&empty_bar[stage], phase ^ 1);
        mbar_expect_tx(&full_bar[stage], WG_STAGE);
        uint8_t* sa = smem + stage * WG_STAGE;
#pragma unroll
        for (int b = 0; b < 2; ++b) {
          const int u = b ? u1 : u0;
          const int ti = u / p.c_blocks, cb = u - ti * p.c_blocks;
          const Tap t = p.taps[ti];
          const bool first = cb < p.c0_blocks;
          const CUtensorMap* ma = first ? &mapA0 : &mapA1;
          const int cch = (first ? cb : cb - p.c0_blocks) * 64;
          if (!p.s2) tma_load_4d(sa + b * WG_BLK, ma, &full_bar[stage], cch, x0 + t.dx, y0 + t.dy, n0);
          else tma_load_5d(sa + b * WG_BLK, ma, &full_bar[stage], t.px * p.c0 + cch, x0 + t.dx, t.py, y0 + t.dy, n0);
        }
#pragma unroll
        for (int j = 0; j < WG_N / 64; ++j)
          tma_load_4d(sa + (2 + j) * WG_BLK, &mapG, &full_bar[stage], nt * WG_N + j * 64, x0, y0, n0);
        if (++stage == WG_STAGES) { stage = 0; phase ^= 1; }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      constexpr uint32_t idesc128 = idesc_bf16(128, 128, 1, 1), idesc192 = idesc_bf16(128, 192, 1, 1);
      constexpr uint64_t dbase = smem_desc_sw128(WG_BLK, 1024);      // MN-major: LBO = next 64-channel block
      int stage = 0; uint32_t phase = 0, tphase = 0;
      bool fresh = true;
      for (long long w = wb; w < we; ++w) {
        const int pt = (int)(w % p.pix_tiles);
        if (fresh) {                       // new output tile: the epilogue must have drained the accumulator
          mbar_wait(&tempty_bar, tphase ^ 1);
          tc_fence_after();
        }
        mbar_wait(&full_bar[stage], phase);
        tc_fence_after();
        const uint32_t a_addr = smem_u32(smem + stage * WG_STAGE), b_addr = a_addr + 2 * WG_BLK;
#pragma unroll
        for (int k = 0; k < WG_PIX / 16; ++k) {
          const uint32_t acc = (!fresh || k != 0);
          const uint64_t da = desc_with_addr(dbase, a_addr + k * 2048);
          umma_bf16(tmem_base, da, desc_with_addr(dbase, b_addr + k * 2048), idesc128, acc);
          umma_bf16(tmem_base + 128, da, desc_with_addr(dbase, b_addr + 2 * WG_BLK + k * 2048), idesc192, acc);
        }
        umma_commit(&empty_bar[stage]);
        if (++stage == WG_STAGES) { stage = 0; phase ^= 1; }
        fresh = false;
        if (pt == p.pix_tiles - 1 || w == we - 1) {      // end of this CTA's share of the output tile
          umma_commit(&tfull_bar);
          tphase ^= 1;
          fresh = true;
        }
      }
    }
  } else {
    const int q = warp & 3;
    const int row = q * 32 + lane;
    uint32_t tphase = 0;
    long long w = wb;
    while (w < we) {
      const int ot = (int)(w / p.pix_tiles);
      const long long seg_end = min(we, (long long)(ot + 1) * p.pix_tiles);
      const int nt = ot % p.n_tiles, mt = ot / p.n_tiles;
      const int u0 = 2 * mt;
      const int u = u0 + (row >> 6);
      const bool valid = u < p.units;
      const int ti = valid ? u / p.c_blocks : 0, cb = valid ? u - ti * p.c_blocks : 0;
      const size_t kidx = (size_t)p.taps[ti].widx * p.ctot + cb * 64 + (row & 63);
      mbar_wait(&tfull_bar, tphase);
      tphase ^= 1;
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16);
#pragma unroll 1
      for (int ch = 0; ch < WG_N / 32; ++ch) {
        uint32_t r[32];
        tmem_ld32(taddr + ch * 32, r);
        tmem_ld_wait();
        if (ch == WG_N / 32 - 1) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(&tempty_bar);
        }
        if (valid) {
          float* dst = p.dw + (size_t)(nt * WG_N + ch * 32) * p.ktot + kidx;
#pragma unroll
          for (int i = 0; i < 32; ++i) atomicAdd(dst + (size_t)i * p.ktot, __uint_as_float(r[i]));
        }
      }
      w = seg_end;
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, 512);
  }
}

}  // namespace

bool wgrad_tc_supported(const WgradArgs& a) {
  if (a.dt != DT_BF16 || a.up2) return false;
  if (a.src.c0 % 64 || a.src.c1 % 64 || a.src.c0 == 0 || a.cout % WG_N) return false;
  if (a.ksize != 1 && a.ksize != 3) return false;
  if (a.stride == 2) {
    if (a.ksize != 3 || a.src.c1 || (a.hin & 1) || (a.win & 1) || a.hout * 2 != a.hin || a.wout * 2 != a.win) return false;
  } else if (a.stride != 1 || a.hout != a.hin || a.wout != a.win) {
    return false;
  }
  int bw, bh, bn;
  return tile_geometry64(a.hout, a.wout, bw, bh, bn);
}

int wgrad_tc(const WgradArgs& a, cudaStream_t st) {
  WgParams p;
  memset(&p, 0, sizeof p);
  const bool s2 = a.stride == 2;
  tile_geometry64(a.hout, a.wout, p.bw, p.bh, p.bn);
  p.c0 = a.src.c0; p.ctot = a.src.c(); p.c0_blocks = a.src.c0 / 64; p.c_blocks = p.ctot / 64; p.s2 = s2;
  const int taps = a.ksize * a.ksize, pad = (a.ksize - 1) / 2;
  p.units = taps * p.c_blocks; p.ktot = taps * p.ctot;
  for (int r = 0; r < a.ksize; ++r)
    for (int s = 0; s < a.ksize; ++s) {
      Tap t; t.widx = r * a.ksize + s; t.px = t.py = 0;
      if (!s2) { t.dy = r - pad; t.dx = s - pad; }
      else { t.dy = r == 0 ? -1 : 0; t.py = r == 1 ? 0 : 1; t.dx = s == 0 ? -1 : 0; t.px = s == 1 ? 0 : 1; }
      p.taps[t.widx] = t;
    }
  p.tiles_w = a.wout / p.bw; p.tiles_h = (a.hout + p.bh - 1) / p.bh;
  p.pix_tiles = p.tiles_w * p.tiles_h * ((a.n + p.bn - 1) / p.bn);
  p.m_tiles = (p.units + 1) / 2; p.n_tiles = a.cout / WG_N;
  p.dw = a.dw;
  CUtensorMap m0, m1, mg;
  bool ok;
  if (s2) ok = act_map_s2(a.src.p0, a.n, a.hin, a.win, a.src.c0, p.bw, p.bh, p.bn, &m0);
  else ok = act_map(a.src.p0, a.n, a.hin, a.win, a.src.c0, p.bw, p.bh, p.bn, &m0);
  m1 = m0;
  if (ok && a.src.c1) ok = act_map(a.src.p1, a.n, a.hin, a.win, a.src.c1, p.bw, p.bh, p.bn, &m1);
  if (ok) ok = act_map(a.g, a.n, a.hout, a.wout, a.cout, p.bw, p.bh, p.bn, &mg);
  if (!ok) return -1;
  static bool attr_set = false;
  if (!attr_set) {
    if (cudaFuncSetAttribute(wgrad_tc_k, cudaFuncAttributeMaxDynamicSharedMemorySize, WG_SMEM) != cudaSuccess) {
      tmap::set_error("cudaFuncSetAttribute(wgrad smem) failed");
      return -1;
    }
    attr_set = true;
  }
  p.work = (long long)p.m_tiles * p.n_tiles * p.pix_tiles;
  // one CTA per SM, each with an equal share of the work items (at least 4 per CTA)
  long long ctas = sm_count();
  if (p.work / 4 < ctas) ctas = p.work / 4 > 0 ? p.work / 4 : 1;
  wgrad_tc_k<<<(unsigned)ctas, 192, WG_SMEM, st>>>(m0, m1, mg, p);
  return 1;
}

}  // namespace pulse

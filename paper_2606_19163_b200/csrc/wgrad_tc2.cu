// wgrad_tc2.cu - CTA-pair (tcgen05 cta_group::2) weight-gradient kernel for sm_100a.
//   dW[co][tap][c] += sum_pixels g[pixel, co] * in[pixel shifted by tap, c]
// GEMM view: D[256 rows = 4 x (tap, 64-channel block)][320 cols = co] += A^T B over K = pixels.  Both operands
// have the channel dimension contiguous (MN-major), so the fprop TMA boxes ([64 pixels][64 channels], 128-byte
// swizzled rows) are consumed directly by MN-major UMMA descriptors.
// Pair tile: each CTA loads ITS two (tap, channel-block) units of the activations (16 KB) and HALF of the
// gradient columns (co): 128 of the first 256 (two 64-wide boxes) and 32 of the last 64 (one 64-byte-swizzled
// box) = 20 KB, and the leader issues M = 256 MMAs with N = 256 and N = 64.  Per CTA that is 36 KB of operands
// per 640 MMA cycles (the single-CTA kernel moves 56 KB for the same math and is bound by shared-memory
// bandwidth: TMA writes + MMA reads > 128 B/cycle/SM).
// Work distribution ("stream-K"): items (output tile, 64-pixel tile) are cut into equal contiguous ranges, one
// per CTA pair; a range that crosses an output-tile boundary flushes its accumulator with fp32 red.add into dW
// (which is also how weight gradients accumulate across microbatches, row a11) and starts the next tile.
#include <cuda.h>

#include <cstdlib>
#include <cstring>

#include "common.cuh"
#include "kernels.h"
#include "sm100.cuh"
#include "tmap.h"

namespace pulse {

namespace {

using namespace sm100;
using namespace tmap;

constexpr int PIX = 64;                       // K per stage
constexpr int BLK = PIX * 128;                // one [64 px][64 ch] box = 8 KB
constexpr int BLK32 = PIX * 64;               // one [64 px][32 ch] box = 4 KB
constexpr int N_TOT = 320;
constexpr int STAGE = 2 * BLK + 2 * BLK + BLK32;      // 36 KB per CTA
constexpr int STAGES = 5;
constexpr int FLUSH_BYTES = 8 * 2 * 2048;             // per epilogue warp: 2 x [16 co][32 c] fp32 boxes
constexpr int SMEM = STAGES * STAGE + FLUSH_BYTES + 1024;

struct Wg2Params {
  int units, c_blocks, c0_blocks, c0, ctot, ktot, s2;
  int up2, gc;                           // up2: the conv of CONV_UP2 (kernels.h): units = (phase, tap, channel block), the
                                         // gradient is read through its parity view (gc = its channel count)
  Tap taps[9];
  int bw, bh, bn, tiles_w, tiles_h;
  int pix_tiles, m_tiles, n_tiles;       // m_tiles: pair tiles of 4 units
  long long work;
  int ppt;                               // pairs per output tile (aligned split) or 0 (stream-K)
  int whole, store;                      // whole: every output tile belongs to one pair (contiguous runs of tiles); store: plain stores
  float* dw;
};

template <bool UP2>      // compile-time: the plain conv's kernel carries none of the phase-form code
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(320, 1)
wgrad_tc2_k(const __grid_constant__ CUtensorMap mapA0, const __grid_constant__ CUtensorMap mapA1,
            const __grid_constant__ CUtensorMap mapG, const __grid_constant__ CUtensorMap mapG32,
            const __grid_constant__ CUtensorMap mapW, const Wg2Params p) {
  extern __shared__ uint8_t smem_raw[];
  __shared__ uint64_t full_bar[STAGES], empty_bar[STAGES], tfull_bar, tempty_bar;
  __shared__ uint32_t tmem_base_s;
  uint8_t* smem = smem_raw + ((1024 - (smem_u32(smem_raw) & 1023)) & 1023);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int pair = blockIdx.x >> 1, npairs = gridDim.x >> 1;
  // ranges: aligned (ppt pairs per output tile, each a share of its pixel tiles: one flush per pair) when there are
  // at least as many pairs as output tiles, else equal contiguous ranges over everything (stream-K)
  long long wb, we;
  if (p.ppt > 0) {
    const int ot = pair / p.ppt, k = pair - ot * p.ppt;
    wb = (long long)ot * p.pix_tiles + (long long)p.pix_tiles * k / p.ppt;
    we = (long long)ot * p.pix_tiles + (long long)p.pix_tiles * (k + 1) / p.ppt;
  } else if (p.whole) {
    const long long tiles = (long long)p.m_tiles * p.n_tiles;
    wb = tiles * pair / npairs * p.pix_tiles; we = tiles * (pair + 1) / npairs * p.pix_tiles;
  } else {
    wb = p.work * pair / npairs; we = p.work * (pair + 1) / npairs;
  }

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&mapA0); prefetch_tmap(&mapA1); prefetch_tmap(&mapG); prefetch_tmap(&mapG32); prefetch_tmap(&mapW);
    for (int i = 0; i < STAGES; ++i) { mbar_init(&full_bar[i], 1); mbar_init(&empty_bar[i], 1); }
    mbar_init(&tfull_bar, 1); mbar_init(&tempty_bar, 16);
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc2(&tmem_base_s, 512);
  tc_fence_before();
  cluster_sync_all();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_s;
  pdl_wait();
  pdl_launch_dependents();

  if (warp == 0) {
    if (lane == 0) {
      // ===== TMA producer (both CTAs) =====
      // indices advance incrementally: a 64-bit division per work item would cost more than the item's MMAs
      int stage = 0; uint32_t phase = 0;
      int ot = (int)(wb / p.pix_tiles), pt = (int)(wb - (long long)ot * p.pix_tiles);
      int tx = pt % p.tiles_w, ty = (pt / p.tiles_w) % p.tiles_h, tn = pt / (p.tiles_w * p.tiles_h);
      const int n_items = (int)(we - wb);
      const CUtensorMap* ma[2]; int cch[2], adx[2], ady[2], apx[2], apy[2], co = 0, gpx = 0, gpy = 0;
      bool new_tile = true;
      for (int it = 0; it < n_items; ++it) {
        if (new_tile) {
          const int nt = ot % p.n_tiles, mt = ot / p.n_tiles;
#pragma unroll
          for (int b = 0; b < 2; ++b) {
            const int u = min(4 * mt + 2 * (int)rank + b, p.units - 1);
            const int ti = u / p.c_blocks, cb = u - ti * p.c_blocks;
            const bool first = cb < p.c0_blocks;
            ma[b] = first ? &mapA0 : &mapA1;
            cch[b] = (first ? cb : cb - p.c0_blocks) * 64;
            if (!UP2) {
              const Tap t = p.taps[ti];
              adx[b] = t.dx; ady[b] = t.dy; apx[b] = t.px; apy[b] = t.py;
            } else {      // ti = 4 (2 py + px) + 2 a + b': low-resolution pixel (y + a - 1 + py, x + b' - 1 + px)
              gpy = ti >> 3; gpx = (ti >> 2) & 1;
              ady[b] = ((ti >> 1) & 1) - 1 + gpy; adx[b] = (ti & 1) - 1 + gpx; apx[b] = apy[b] = 0;
            }
          }
          co = nt * N_TOT;
          new_tile = false;
        }
        const int x0 = tx * p.bw, y0 = ty * p.bh, n0 = tn * p.bn;
        mbar_wait(&empty_bar[stage], phase ^ 1);
        {
          if (rank == 0) mbar_expect_tx(&full_bar[stage], 2 * STAGE);
          const uint32_t fb = mapa_u32(smem_u32(&full_bar[stage]), 0);
          uint8_t* sa = smem + stage * STAGE;
#pragma unroll
          for (int b = 0; b < 2; ++b) {
            if (!p.s2) tma2_load_4d(sa + b * BLK, ma[b], fb, cch[b], x0 + adx[b], y0 + ady[b], n0);
            else tma2_load_5d(sa + b * BLK, ma[b], fb, apx[b] * p.c0 + cch[b], x0 + adx[b], apy[b], y0 + ady[b], n0);
          }
          if (!UP2) {
            tma2_load_4d(sa + 2 * BLK, &mapG, fb, co + (int)rank * 128, x0, y0, n0);
            tma2_load_4d(sa + 3 * BLK, &mapG, fb, co + (int)rank * 128 + 64, x0, y0, n0);
            tma2_load_4d(sa + 4 * BLK, &mapG32, fb, co + 256 + (int)rank * 32, x0, y0, n0);
          } else {        // the pixels (2y + py, 2x + px) of the gradient: parity view (px gc + channel, x, py, y, n)
            const int gco = gpx * p.gc + co;
            tma2_load_5d(sa + 2 * BLK, &mapG, fb, gco + (int)rank * 128, x0, gpy, y0, n0);
            tma2_load_5d(sa + 3 * BLK, &mapG, fb, gco + (int)rank * 128 + 64, x0, gpy, y0, n0);
            tma2_load_5d(sa + 4 * BLK, &mapG32, fb, gco + 256 + (int)rank * 32, x0, gpy, y0, n0);
          }
        }
        if (++stage == STAGES) { stage = 0; phase ^= 1; }
        if (++tx == p.tiles_w) { tx = 0; if (++ty == p.tiles_h) { ty = 0; ++tn; } }
        if (++pt == p.pix_tiles) { pt = 0; tx = ty = tn = 0; ++ot; new_tile = true; }
      }
    }
  } else if (warp == 1) {
    if (rank == 0) {
      // ===== MMA issuer (leader): the whole warp runs the loop, one elected lane issues (see elect_one_sync) =====
      constexpr uint32_t idesc256 = idesc_bf16(256, 256, 1, 1), idesc64 = idesc_bf16(256, 64, 1, 1);
      constexpr uint64_t d128 = smem_desc_sw128(BLK, 1024);      // MN-major: LBO = next 64-channel block, SBO = 8 pixels
      constexpr uint64_t d64 = smem_desc_sw64(BLK32, 512);
      constexpr uint32_t hi128 = (uint32_t)(d128 >> 32), hi64 = (uint32_t)(d64 >> 32);
      const uint32_t base16 = (smem_u32(smem) >> 4) & 0x3FFF;
      int stage = 0; uint32_t phase = 0, tphase = 0;
      bool fresh = true;
      int pt = (int)(wb % p.pix_tiles);
      const int n_items = (int)(we - wb);
      for (int it = 0; it < n_items; ++it) {
        if (fresh) {
          mbar_wait(&tempty_bar, tphase ^ 1);
          tc_fence_after();
        }
        mbar_wait(&full_bar[stage], phase);
        tc_fence_after();
        const uint32_t a16 = base16 + stage * (STAGE >> 4);
        const bool last = (++pt == p.pix_tiles || it == n_items - 1);
        if (elect_one_sync()) {
          {
#pragma unroll
            for (int k = 0; k < PIX / 16; ++k) {
              const uint32_t acc = (!fresh || k != 0);
              const uint64_t da = ((uint64_t)hi128 << 32) | ((uint32_t)d128 | (a16 + k * 128));
              umma2_bf16(tmem_base, da, ((uint64_t)hi128 << 32) | ((uint32_t)d128 | (a16 + (2 * BLK >> 4) + k * 128)),
                         idesc256, acc);
              umma2_bf16(tmem_base + 256, da, ((uint64_t)hi64 << 32) | ((uint32_t)d64 | (a16 + (4 * BLK >> 4) + k * 64)),
                         idesc64, acc);
            }
          }
          umma2_commit_mc(&empty_bar[stage], 3);
          if (last) umma2_commit_mc(&tfull_bar, 3);
        }
        __syncwarp();
        if (++stage == STAGES) { stage = 0; phase ^= 1; }
        fresh = false;
        if (last) { pt = 0; tphase ^= 1; fresh = true; }
      }
    }
  } else {
    // ===== epilogue (both CTAs, warps 2..9): this CTA's 128 rows x 320 columns are ADDED into dW (fp32).  A warp
    // reads 32 consecutive channels c (the TMEM lane quadrant warp % 4); the two warps of a quadrant take alternate
    // 16-column chunks.  Per chunk a warp transposes its registers into a [16 co][32 c] fp32 box in shared memory
    // (conflict-free: a row is one 128-byte line) and one TMA reduce-add instruction replaces 512 scalar atomics;
    // boxes are double-buffered per warp and the TMEM load of the next chunk is issued before the current one is
    // stored.
    const int q = warp & 3, grp = (warp - 2) >> 2;
    uint8_t* stg = smem + STAGES * STAGE + q * 8192 + grp * 4096;
    const uint32_t stg_lane = smem_u32(stg) + lane * 4;
    uint32_t tphase = 0;
    int buf = 0;
    long long w = wb;
    while (w < we) {
      const int ot = (int)(w / p.pix_tiles);
      const long long seg_end = min(we, (long long)(ot + 1) * p.pix_tiles);
      const int nt = ot % p.n_tiles, mt = ot / p.n_tiles;
      const int u = 4 * mt + 2 * (int)rank + (q >> 1);
      const bool valid = u < p.units;
      const int ti = valid ? u / p.c_blocks : 0, cb = valid ? u - ti * p.c_blocks : 0;
      const int kch = cb * 64 + (q & 1) * 32;
      const int kcol = p.taps[UP2 ? 0 : ti].widx * p.ctot + kch;
      // up2: this unit's partial belongs to every (r, s) its pre-summed tap covers: rows r0..r1, columns s0..s1 of the 3x3
      int r0 = 0, r1 = 0, s0 = 0, s1 = 0;
      if (UP2) {
        const int py = ti >> 3, px = (ti >> 2) & 1, ta = (ti >> 1) & 1, tb = ti & 1;
        r0 = (py == 0 && ta == 1) ? 1 : (py == 1 && ta == 1) ? 2 : 0; r1 = (py == 0 && ta == 0) ? 0 : (py == 1 && ta == 0) ? 1 : 2;
        s0 = (px == 0 && tb == 1) ? 1 : (px == 1 && tb == 1) ? 2 : 0; s1 = (px == 0 && tb == 0) ? 0 : (px == 1 && tb == 0) ? 1 : 2;
      }
      mbar_wait(&tfull_bar, tphase);
      tphase ^= 1;
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16);
      constexpr int NIT = N_TOT / 32;          // 20 chunks of 16 columns, 10 per warp
      uint32_t rr[2][16];
      tmem_ld16(taddr + grp * 16, rr[0]);
#pragma unroll
      for (int it = 0; it < NIT; ++it) {
        const int ch = grp + 2 * it;
        uint32_t (&r)[16] = rr[it & 1];
        tmem_ld_wait();
        if (it + 1 < NIT) {
          tmem_ld16(taddr + (ch + 2) * 16, rr[(it + 1) & 1]);
        } else {                                 // that was this warp's last TMEM read of the tile
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster_relaxed(mapa_u32(smem_u32(&tempty_bar), 0));
        }
        if (valid) {
          if (lane == 0) bulk_wait_read<1>();
          __syncwarp();
          const uint32_t dst = stg_lane + buf * 2048;
#pragma unroll
          for (int i = 0; i < 16; ++i) asm volatile("st.shared.b32 [%0], %1;" ::"r"(dst + i * 128), "r"(r[i]) : "memory");
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) {
            if (!UP2) {
              if (p.store) tma_store_2d(&mapW, stg + buf * 2048, kcol, nt * N_TOT + ch * 16);
              else tma_reduce_add_2d(&mapW, stg + buf * 2048, kcol, nt * N_TOT + ch * 16);
            } else {
              for (int r = r0; r <= r1; ++r)
                for (int s_ = s0; s_ <= s1; ++s_)
                  tma_reduce_add_2d(&mapW, stg + buf * 2048, (r * 3 + s_) * p.ctot + kch, nt * N_TOT + ch * 16);
            }
            bulk_commit();
          }
          buf ^= 1;
        }
      }
      w = seg_end;
    }
    if (lane == 0) bulk_wait_read<0>();       // the staging boxes have been read; the reductions complete before the grid does
  }
  tc_fence_before();
  cluster_sync_all();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc2(tmem_base, 512);
  }
}

}  // namespace

bool wgrad_tc2_supported(const WgradArgs& a) {
  if (a.dt != DT_BF16) return false;
  if (a.src.c0 % 64 || a.src.c1 % 64 || a.src.c0 == 0 || a.cout % N_TOT) return false;
  if (a.ksize != 1 && a.ksize != 3) return false;
  int bw, bh, bn;
  if (a.up2) {
    if (a.ksize != 3 || a.src.c1 || a.hout != 2 * a.hin || a.wout != 2 * a.win) return false;
    return tile_geometry64(a.hin, a.win, bw, bh, bn);
  }
  if (a.stride == 2) {
    if (a.ksize != 3 || a.src.c1 || (a.hin & 1) || (a.win & 1) || a.hout * 2 != a.hin || a.wout * 2 != a.win) return false;
  } else if (a.stride != 1 || a.hout != a.hin || a.wout != a.win) {
    return false;
  }
  return tile_geometry64(a.hout, a.wout, bw, bh, bn);
}

// Whole-tile ownership: at least as many output tiles as pairs, and runs of ceil(tiles / pairs) tiles waste at most a
// quarter of the machine.  Then a tile's pixel range is never shared, the flush may STORE (first backward of a step) and
// the 59 - 118 MB gradient of a 1280-channel conv is written once instead of zeroed, read and written.
bool wgrad_whole_tiles(const WgradArgs& a) {
  if (a.up2 || !wgrad_tc2_supported(a) || toggles().wgrad_1cta) return false;
  const long long units = (long long)a.ksize * a.ksize * (a.src.c() / 64);
  const long long tiles = (units + 3) / 4 * (a.cout / N_TOT), pairs = sm_count() / 2;
  return tiles >= pairs && ((tiles + pairs - 1) / pairs) * pairs * 4 <= 5 * tiles;
}

int wgrad_tc2(const WgradArgs& a, cudaStream_t st) {
  Wg2Params p;
  memset(&p, 0, sizeof p);
  const bool s2 = !a.up2 && a.stride == 2;
  const int gh = a.up2 ? a.hin : a.hout, gw = a.up2 ? a.win : a.wout;      // pixel grid of the K dimension
  tile_geometry64(gh, gw, p.bw, p.bh, p.bn);
  p.up2 = a.up2; p.gc = a.cout;
  p.c0 = a.src.c0; p.ctot = a.src.c(); p.c0_blocks = a.src.c0 / 64; p.c_blocks = p.ctot / 64; p.s2 = s2;
  const int taps = a.ksize * a.ksize, pad = (a.ksize - 1) / 2;
  p.units = (a.up2 ? 16 : taps) * p.c_blocks; p.ktot = taps * p.ctot;
  for (int r = 0; r < a.ksize; ++r)
    for (int s = 0; s < a.ksize; ++s) {
      Tap t; t.widx = r * a.ksize + s; t.px = t.py = 0;
      if (!s2) { t.dy = r - pad; t.dx = s - pad; }
      else { t.dy = r == 0 ? -1 : 0; t.py = r == 1 ? 0 : 1; t.dx = s == 0 ? -1 : 0; t.px = s == 1 ? 0 : 1; }
      p.taps[t.widx] = t;
    }
  p.tiles_w = gw / p.bw; p.tiles_h = (gh + p.bh - 1) / p.bh;
  p.pix_tiles = p.tiles_w * p.tiles_h * ((a.n + p.bn - 1) / p.bn);
  p.m_tiles = (p.units + 3) / 4; p.n_tiles = a.cout / N_TOT;
  p.dw = a.dw;
  CUtensorMap m0, m1, mg, mg32, mw;
  bool ok;
  if (s2) ok = act_map_s2(a.src.p0, a.n, a.hin, a.win, a.src.c0, p.bw, p.bh, p.bn, &m0);
  else ok = act_map(a.src.p0, a.n, a.hin, a.win, a.src.c0, p.bw, p.bh, p.bn, &m0);
  m1 = m0;
  if (ok && a.src.c1) ok = act_map(a.src.p1, a.n, a.hin, a.win, a.src.c1, p.bw, p.bh, p.bn, &m1);
  if (ok && !a.up2) ok = act_map(a.g, a.n, a.hout, a.wout, a.cout, p.bw, p.bh, p.bn, &mg);
  if (ok && !a.up2) ok = act_map_c(a.g, a.n, a.hout, a.wout, a.cout, 32, p.bw, p.bh, p.bn, &mg32);
  if (ok && a.up2) ok = act_map_s2(a.g, a.n, a.hout, a.wout, a.cout, p.bw, p.bh, p.bn, &mg);
  if (ok && a.up2) ok = act_map_s2_c(a.g, a.n, a.hout, a.wout, a.cout, 32, p.bw, p.bh, p.bn, &mg32);
  if (ok) ok = mat_map_f32(a.dw, a.cout, p.ktot, 32, 16, &mw);
  if (!ok) return -1;
  static bool attr_set = false;
  if (!attr_set) {
    if (cudaFuncSetAttribute(wgrad_tc2_k<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM) != cudaSuccess ||
        cudaFuncSetAttribute(wgrad_tc2_k<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM) != cudaSuccess) {
      tmap::set_error("cudaFuncSetAttribute(wgrad2 smem) failed");
      return -1;
    }
    attr_set = true;
  }
  p.work = (long long)p.m_tiles * p.n_tiles * p.pix_tiles;
  long long pairs = sm_count() / 2;                       // one CTA pair per SM pair, equal shares, >= 4 items each
  if (p.work / 4 < pairs) pairs = p.work / 4 > 0 ? p.work / 4 : 1;
  const long long out_tiles = (long long)p.m_tiles * p.n_tiles;
  p.ppt = 0;
  p.whole = wgrad_whole_tiles(a); p.store = p.whole && a.overwrite;
  if (p.whole) pairs = sm_count() / 2;
  if (out_tiles <= pairs && p.pix_tiles >= 4 * (pairs / out_tiles)) {       // aligned split: one flush per pair
    p.ppt = (int)(pairs / out_tiles);
    pairs = p.ppt * out_tiles;
  }
  if (a.up2) launch_pdl(wgrad_tc2_k<true>, dim3((unsigned)(2 * pairs)), dim3(320), SMEM, st, m0, m1, mg, mg32, mw, p);
  else launch_pdl(wgrad_tc2_k<false>, dim3((unsigned)(2 * pairs)), dim3(320), SMEM, st, m0, m1, mg, mg32, mw, p);
  return 1;
}

static bool force_1cta_wgrad() { return toggles().wgrad_1cta; }
bool wgrad_tc_any_supported(const WgradArgs& a) { return wgrad_tc2_supported(a) || wgrad_tc_supported(a); }
int wgrad_tc_any(const WgradArgs& a, cudaStream_t st) {
  if ((!force_1cta_wgrad() || a.up2) && wgrad_tc2_supported(a)) return wgrad_tc2(a, st);
  return wgrad_tc(a, st);
}

}  // namespace pulse

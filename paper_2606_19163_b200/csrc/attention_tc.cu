// attention_tc.cu - tcgen05 forward of the attention core for bf16 tensors with 64 or 128 channels per head
// (formulas in attention.cu).  One CTA = 128 queries of one (image, head); query row i = TMEM lane i
// is shared by the two threads i and 128 + i (warps w and w + 4 reach the same lane quadrant), each taking half of the
// columns, so the softmax needs one exchange of the row maximum / sum per sweep and no shuffles:
//   sweep 1 over the key tiles:  S = Q K^T (tcgen05.mma, M = 128, N = 128, K = d, both operands K-major from TMA boxes
//                                of the interleaved qkv tensor) -> TMEM -> row maximum m_i
//   sweep 2:                     S again -> p = 2^((s - m_i) scale log2 e) -> l_i += p, P as bf16 into a 128-byte-swizzled
//                                A-operand tile -> O += P V (V is read MN-major, straight from its [keys][d] box) in TMEM
//   epilogue:                    o_i = O_i / l_i -> bf16 -> global; log-sum-exp_i = m_i scale + ln l_i for the backward.
// Roles: warps 0-7 are the softmax threads; warp 8 issues every TMA load and MMA.  The S columns are copied to registers
// in one go and released (bar_sfree), so the Q K^T of the NEXT key tile runs on the tensor pipe while the exponentials of
// this one are computed; P V of this tile is queued behind it.  K tiles are double-buffered, V is refilled as soon as its
// P V has completed.  96 KB of shared memory and 256 TMEM columns: two CTAs per SM.
// Two sweeps instead of the online rescale: O lives in tensor memory, where a rescale per key tile would cost a TMEM
// round trip of the whole accumulator; the second Q K^T is 1/3 more MMA work on a kernel whose bound is the exponential
// (128 x 128 MUFU ops per tile = 1024 cycles against 512 of MMA).
#include <cuda.h>

#include "common.cuh"
#include "kernels.h"
#include "sm100.cuh"
#include "tmap.h"

namespace pulse {

namespace {

using namespace sm100;

constexpr int BQ = 128, BKEY = 128;
constexpr int CH = BQ * 128;                    // one [128 rows][64 bf16] chunk: 16 KB

template <int D> struct ACfg {
  static constexpr int NC = D / 64;             // 64-channel chunks per row
  static constexpr int KV_BYTES = NC * CH;                      // one K tile
  // Q | K double-buffered | V | P: 96 KB at d = 64, so that two CTAs share an SM
  static constexpr int Q_OFF = 0, KV_OFF = NC * CH, V_OFF = 3 * NC * CH, P_OFF = 4 * NC * CH;
  static constexpr int SMEM = 4 * NC * CH + 2 * CH + 1024;
  static constexpr int TMEM_COLS = 256;         // S: columns [0, 128), O: [128, 128 + D)
};

struct AtcP { int T, C, heads; float scale; bf16* o; float* lse; };

// 2^x for x <= 0 (scores minus their row maximum / log-sum-exp): one MUFU.EX2; results below 2^-126 flush to zero, which
// exp2f() would pay a compare and two multiplies per element to keep
__device__ __forceinline__ float ex2a(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

// all three kernels: warps 0-7 = softmax (two per TMEM lane quadrant), warp 8 = TMA + MMA issue
constexpr int SOFTMAX_THREADS = 256, ISSUER_WARP = 8, FWD_THREADS = SOFTMAX_THREADS + 32;
__device__ __forceinline__ void softmax_sync() { asm volatile("bar.sync 1, %0;" ::"n"(SOFTMAX_THREADS) : "memory"); }

template <int D>
__global__ void __launch_bounds__(FWD_THREADS, 2) attn_fwd_tc_k(const __grid_constant__ CUtensorMap map, const AtcP p) {
  using A = ACfg<D>;
  extern __shared__ uint8_t smem_raw[];
  // bar_s: S = Q K^T complete | bar_sfree: all softmax threads hold their S columns in registers | bar_p: P written |
  // bar_pv: O += P V complete (P and the V tile are free)
  __shared__ uint64_t bar_q, bar_k[2], bar_v, bar_s, bar_sfree, bar_p, bar_pv;
  __shared__ uint32_t tmem_base_s;
  __shared__ float xch[2][2][BQ];            // [m | l, lx][column half][row]
  uint8_t* smem = smem_raw + ((1024 - (smem_u32(smem_raw) & 1023)) & 1023);
  const int warp = threadIdx.x >> 5;
  const int q0 = blockIdx.x * BQ, h = blockIdx.y, n = blockIdx.z;
  const int nkb = (p.T + BKEY - 1) / BKEY, nit = 2 * nkb;
  if (threadIdx.x == 0) {
    prefetch_tmap(&map);
    mbar_init(&bar_q, 1); mbar_init(&bar_k[0], 1); mbar_init(&bar_k[1], 1); mbar_init(&bar_v, 1);
    mbar_init(&bar_s, 1); mbar_init(&bar_sfree, SOFTMAX_THREADS); mbar_init(&bar_p, SOFTMAX_THREADS); mbar_init(&bar_pv, 1);
    fence_barrier_init();
  }
  if (warp == ISSUER_WARP) tmem_alloc(&tmem_base_s, A::TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_base_s;
  pdl_wait();
  pdl_launch_dependents();
  const uint32_t sb = smem_u32(smem);

  if (warp == ISSUER_WARP) {
    // ---------------------------------------------------------------- TMA + MMA issue (whole warp runs the loop, one lane issues)
    constexpr uint64_t dk = smem_desc_sw128(16, 1024);            // K-major operand: 128-byte rows, 8-row atoms
    constexpr uint64_t dmn = smem_desc_sw128(CH, 1024);           // MN-major operand (V): LBO = next 64-channel chunk
    constexpr uint32_t idesc_s = idesc_bf16(BQ, BKEY, 0, 0), idesc_o = idesc_bf16(BQ, D, 0, 1);
    // K tiles are double-buffered over the 2 nkb iterations of the two sweeps; V has one buffer, refilled as soon as the
    // P V product that read it has completed
    auto load_k = [&](int it) {
      const int b = it & 1, kb = it % nkb;
      if (elect_one_sync()) {
        mbar_expect_tx(&bar_k[b], A::NC * CH);
        for (int c = 0; c < A::NC; ++c)
          tma_load_3d(smem + A::KV_OFF + b * A::KV_BYTES + c * CH, &map, &bar_k[b], p.C + h * D + 64 * c, kb * BKEY, n);
      }
    };
    auto load_v = [&](int kb) {
      if (elect_one_sync()) {
        mbar_expect_tx(&bar_v, A::NC * CH);
        for (int c = 0; c < A::NC; ++c)
          tma_load_3d(smem + A::V_OFF + c * CH, &map, &bar_v, 2 * p.C + h * D + 64 * c, kb * BKEY, n);
      }
    };
    auto issue_pv = [&](int j) {                                  // j: key tile of sweep 2
      mbar_wait(&bar_p, j & 1);
      mbar_wait(&bar_v, j & 1);
      tc_fence_after();
#pragma unroll
      for (int k = 0; k < BKEY / 16; ++k) {
        const uint32_t pa = sb + A::P_OFF + (k / 4) * CH + (k % 4) * 32;      // A = P, K-major: keys 16 k ..
        const uint32_t vb = sb + A::V_OFF + k * 2048;                         // B = V, MN-major: 16 key rows of 128 bytes
        if (elect_one_sync()) umma_bf16(tmem + 128, desc_with_addr(dk, pa), desc_with_addr(dmn, vb), idesc_o, (j | k) != 0);
      }
      if (elect_one_sync()) umma_commit(&bar_pv);
      __syncwarp();
    };
    if (elect_one_sync()) {
      mbar_expect_tx(&bar_q, A::NC * CH);
      for (int c = 0; c < A::NC; ++c) tma_load_3d(smem + A::Q_OFF + c * CH, &map, &bar_q, h * D + 64 * c, q0, n);
    }
    load_k(0);
    mbar_wait(&bar_q, 0);
    for (int it = 0; it < nit; ++it) {
      const int b = it & 1;
      mbar_wait(&bar_k[b], (it >> 1) & 1);
      if (it > 0) mbar_wait(&bar_sfree, (it - 1) & 1);           // S(it - 1) is in registers (and its MMA done: K buffer b ^ 1 free)
      tc_fence_after();
#pragma unroll
      for (int k = 0; k < D / 16; ++k) {                          // S = Q K^T: runs while the softmax threads work on S(it - 1)
        const uint32_t off = (k / 4) * CH + (k % 4) * 32;        // chunk of 64 channels, 32 bytes per K = 16 step
        if (elect_one_sync())
          umma_bf16(tmem, desc_with_addr(dk, sb + A::Q_OFF + off), desc_with_addr(dk, sb + A::KV_OFF + b * A::KV_BYTES + off), idesc_s, k != 0);
      }
      if (elect_one_sync()) umma_commit(&bar_s);
      __syncwarp();
      if (it + 1 < nit) load_k(it + 1);
      if (it > nkb) issue_pv(it - 1 - nkb);                       // O += P V of the previous sweep-2 tile, behind S(it) in the pipe
      if (it >= nkb) {
        if (it > nkb) mbar_wait(&bar_pv, (it - 1 - nkb) & 1);    // V's reader has completed
        load_v(it - nkb);
      }
    }
    issue_pv(nkb - 1);
  } else {
    // ---------------------------------------------------------------- softmax: thread = (query row, half of the key columns)
    const int row = threadIdx.x & (BQ - 1), half = threadIdx.x >> 7;
    const uint32_t trow = tmem + ((uint32_t)((warp & 3) * 32) << 16);
    const float c2 = p.scale * 1.4426950408889634f;
    float m = -INFINITY, l = 0.f, lx = 0.f, mc = 0.f;    // l: sum of the bf16 probabilities the P V product sees; lx: the exact sum
    for (int it = 0; it < nit; ++it) {
      const int kb = it % nkb;
      if (it == nkb) {                     // between the sweeps: the row maximum of the two column halves
        xch[0][half][row] = m;
        softmax_sync();
        m = fmaxf(xch[0][0][row], xch[0][1][row]);
        mc = m * c2;
      }
      mbar_wait(&bar_s, it & 1);
      tc_fence_after();
      uint32_t r0[32], r1[32];
      tmem_ld32(trow + (2 * half) * 32, r0);
      tmem_ld32(trow + (2 * half + 1) * 32, r1);
      tmem_ld_wait();
      tc_fence_before();
      mbar_arrive(&bar_sfree);             // the next S may overwrite the columns
      const int kbase = kb * BKEY + 2 * half * 32;
      const bool ragged = (kb + 1) * BKEY > p.T;                 // only the last key tile masks its columns
      if (it < nkb) {
        // ---- sweep 1: row maxima of the raw scores
        if (!ragged) {
#pragma unroll
          for (int i = 0; i < 32; ++i) m = fmaxf(m, fmaxf(__uint_as_float(r0[i]), __uint_as_float(r1[i])));
        } else {
#pragma unroll
          for (int i = 0; i < 32; ++i) {
            if (kbase + i < p.T) m = fmaxf(m, __uint_as_float(r0[i]));
            if (kbase + 32 + i < p.T) m = fmaxf(m, __uint_as_float(r1[i]));
          }
        }
        continue;
      }
      // ---- sweep 2: P = exp(scale (S - m)) as bf16 into the A tile
      // o is normalised by the sum of the values the P V product sees (bf16): the rows of P / l sum to one; the
      // log-sum-exp handed to the backward, which recomputes P in fp32, takes the exact sum
      uint32_t pk0[16], pk1[16];
      if (!ragged) {
        // packed fp32 pairs (FFMA2 / FADD2: one issue slot per two keys) around the per-lane MUFU.EX2
        const f2_t c22 = pk2(c2, c2), mc2 = pk2(-mc, -mc);
        f2_t l2 = pk2(l, 0.f), lx2 = pk2(lx, 0.f);
#pragma unroll
        for (int i = 0; i < 32; i += 2) {
          float a0, a1;
          upk2(fma2(pk2(__uint_as_float(r0[i]), __uint_as_float(r0[i + 1])), c22, mc2), a0, a1);
          float e0 = ex2a(a0), e1 = ex2a(a1);
          pk0[i >> 1] = pack_bf16(e0, e1);
          l2 = add2(l2, bf2(pk0[i >> 1]));
          lx2 = add2(lx2, pk2(e0, e1));
          upk2(fma2(pk2(__uint_as_float(r1[i]), __uint_as_float(r1[i + 1])), c22, mc2), a0, a1);
          e0 = ex2a(a0), e1 = ex2a(a1);
          pk1[i >> 1] = pack_bf16(e0, e1);
          l2 = add2(l2, bf2(pk1[i >> 1]));
          lx2 = add2(lx2, pk2(e0, e1));
        }
        float t0, t1;
        upk2(l2, t0, t1); l = t0 + t1;
        upk2(lx2, t0, t1); lx = t0 + t1;
      } else {
#pragma unroll
        for (int i = 0; i < 32; i += 2) {
          float e0 = kbase + i < p.T ? ex2a(fmaf(__uint_as_float(r0[i]), c2, -mc)) : 0.f;
          float e1 = kbase + i + 1 < p.T ? ex2a(fmaf(__uint_as_float(r0[i + 1]), c2, -mc)) : 0.f;
          pk0[i >> 1] = pack_bf16(e0, e1);
          l += __uint_as_float(pk0[i >> 1] << 16) + __uint_as_float(pk0[i >> 1] & 0xffff0000u);
          lx += e0 + e1;
          e0 = kbase + 32 + i < p.T ? ex2a(fmaf(__uint_as_float(r1[i]), c2, -mc)) : 0.f;
          e1 = kbase + 32 + i + 1 < p.T ? ex2a(fmaf(__uint_as_float(r1[i + 1]), c2, -mc)) : 0.f;
          pk1[i >> 1] = pack_bf16(e0, e1);
          l += __uint_as_float(pk1[i >> 1] << 16) + __uint_as_float(pk1[i >> 1] & 0xffff0000u);
          lx += e0 + e1;
        }
      }
      if (it > nkb) mbar_wait(&bar_pv, (it - 1 - nkb) & 1);      // the previous P V has read P
      // keys [32 ch, 32 ch + 32) = 16-byte pieces 4 (ch & 1) .. + 3 of chunk ch / 2 (= half), row `row`, 128-byte swizzle
      const uint32_t base = sb + A::P_OFF + half * CH + row * 128;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        st_shared_v4(base + ((j ^ (row & 7)) << 4), pk0[4 * j], pk0[4 * j + 1], pk0[4 * j + 2], pk0[4 * j + 3]);
        st_shared_v4(base + (((4 + j) ^ (row & 7)) << 4), pk1[4 * j], pk1[4 * j + 1], pk1[4 * j + 2], pk1[4 * j + 3]);
      }
      fence_proxy_async_smem();            // P (generic-proxy writes) before the MMA (async proxy) reads it
      mbar_arrive(&bar_p);
    }
    xch[1][half][row] = l;
    xch[0][half][row] = lx;               // (the maxima have been consumed)
    softmax_sync();
    l = xch[1][0][row] + xch[1][1][row];
    lx = xch[0][0][row] + xch[0][1][row];
    mbar_wait(&bar_pv, (nkb - 1) & 1);
    tc_fence_after();
    // ---- epilogue: o = O / l; each of the row's two threads stores half of the D channels
    const int q = q0 + row;
    const float inv = 1.0f / l;
    bf16* op = p.o + ((size_t)n * p.T + q) * p.C + (size_t)h * D;
#pragma unroll
    for (int cc = 0; cc < D / 64; ++cc) {
      const int ch = half * (D / 64) + cc;
      uint32_t r[32];
      tmem_ld32(trow + 128 + ch * 32, r);
      tmem_ld_wait();
      if (q < p.T) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          uint4 v;
          v.x = pack_bf16(__uint_as_float(r[8 * j]) * inv, __uint_as_float(r[8 * j + 1]) * inv);
          v.y = pack_bf16(__uint_as_float(r[8 * j + 2]) * inv, __uint_as_float(r[8 * j + 3]) * inv);
          v.z = pack_bf16(__uint_as_float(r[8 * j + 4]) * inv, __uint_as_float(r[8 * j + 5]) * inv);
          v.w = pack_bf16(__uint_as_float(r[8 * j + 6]) * inv, __uint_as_float(r[8 * j + 7]) * inv);
          *reinterpret_cast<uint4*>(op + ch * 32 + 8 * j) = v;
        }
      }
    }
    if (q < p.T && half == 0) p.lse[((size_t)n * p.heads + h) * p.T + q] = m * p.scale + __logf(lx);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == ISSUER_WARP) {
    tc_fence_after();
    tmem_dealloc(tmem, A::TMEM_COLS);
  }
}

// ------------------------------------------------------------------------------------------------ backward
// Operand layouts (all tiles are TMA boxes / register-written tiles of 128 rows x 64 bf16 = 128-byte-swizzled chunks):
//   S  = Q K^T, g_P = g_o V^T        A = Q / g_o   K-major,   B = K / V     K-major     (rows = queries, K = channels)
//   g_q += g_S K                     A = g_S       K-major,   B = K         MN-major    (K = keys)
//   g_v += P^T g_o, g_k += g_S^T Q   A = P / g_S   MN-major (their [query][key] tiles read transposed), B = g_o / Q MN-major
// P and g_S are recomputed per tile from the saved log-sum-exp, in fp32 on the TMEM rows (thread = query), and handed to
// the tensor cores as bf16.  D_i = sum_j P_ij g_P_ij comes from a first sweep of the g_q kernel (fp32, from the unrounded
// P: see attention.cu) and is read by the g_k / g_v kernel.
// Roles as in the forward: warps 0-7 recompute P / g_S on the TMEM rows, warp 8 issues every TMA load and MMA.  S and g_P
// go to registers in one pass (4 x tcgen05.ld of 32 columns) and are released at once, so the next tile's S / g_P products
// run while this tile's exponentials are computed, and this tile's accumulating products are queued behind them.  The
// streamed operand tiles go round three buffers at d = 64 (the refill then waits for a product issued one iteration
// earlier, never for one just issued).  Rows / keys past the end need no masks in the g_k / g_v kernel: TMA zero-fills
// them and a zero row of Q, g_o, K or V contributes nothing to any product.
struct AtbP { int T, C, heads; float scale; bf16* g_qkv; const float* lse; float* Dg; };

// 128 fp32 values of this thread's row -> bf16 -> chunk-swizzled A tile at `tile` (two 16 KB chunks of 64 columns)
__device__ __forceinline__ void store_row_chunk32(uint32_t tile, int row, int ch, const uint32_t (&pk)[16]) {
  const uint32_t base = tile + (ch >> 1) * CH + row * 128;
#pragma unroll
  for (int j = 0; j < 4; ++j)
    st_shared_v4(base + ((((ch & 1) * 4 + j) ^ (row & 7)) << 4), pk[4 * j], pk[4 * j + 1], pk[4 * j + 2], pk[4 * j + 3]);
}

template <int D> struct BCfg {
  static constexpr int NC = D / 64;
  static constexpr int PAIR = 2 * NC * CH;                      // two operand tiles (K + V, or Q + g_o)
  // g_q kernel: Q, g_o (resident) | K, V per key tile in NKV buffers | g_S
  static constexpr int NKV = D == 64 ? 3 : 2;
  static constexpr int Q_OFF = 0, GO_OFF = NC * CH, KV_OFF = PAIR, DS_OFF = (1 + NKV) * PAIR;
  static constexpr int SMEM_DQ = (1 + NKV) * PAIR + 2 * CH + 1024;
  // g_k / g_v kernel: K, V (resident) | Q, g_o per query tile in NQB buffers | P, g_S
  static constexpr int NQB = D == 64 ? 3 : 1;
  static constexpr int K_OFF = 0, V_OFF = NC * CH, QG_OFF = PAIR, P_OFF = (1 + NQB) * PAIR, DS2_OFF = (1 + NQB) * PAIR + 2 * CH;
  static constexpr int SMEM_DKV = (1 + NQB) * PAIR + 4 * CH + 1024;
};

template <int D>
__global__ void __launch_bounds__(FWD_THREADS, 1) attn_bwd_dq_tc_k(const __grid_constant__ CUtensorMap mapQ,
                                                                   const __grid_constant__ CUtensorMap mapG, const AtbP p) {
  using B = BCfg<D>;
  extern __shared__ uint8_t smem_raw[];
  // bar_s: S and g_P complete | bar_sfree: both are in the softmax threads' registers | bar_ds: g_S written |
  // bar_dq: g_q += g_S K complete (g_S and that K tile are free)
  __shared__ uint64_t bar_q, bar_kv[B::NKV], bar_s, bar_sfree, bar_ds, bar_dq;
  __shared__ uint32_t tmem_base_s;
  __shared__ float xch[2][BQ];
  uint8_t* smem = smem_raw + ((1024 - (smem_u32(smem_raw) & 1023)) & 1023);
  const int warp = threadIdx.x >> 5;
  const int q0 = blockIdx.x * BQ, h = blockIdx.y, n = blockIdx.z;
  const int nkb = (p.T + BKEY - 1) / BKEY, nit = 2 * nkb;
  if (threadIdx.x == 0) {
    prefetch_tmap(&mapQ); prefetch_tmap(&mapG);
    mbar_init(&bar_q, 1);
    for (int b = 0; b < B::NKV; ++b) mbar_init(&bar_kv[b], 1);
    mbar_init(&bar_s, 1); mbar_init(&bar_sfree, SOFTMAX_THREADS); mbar_init(&bar_ds, SOFTMAX_THREADS); mbar_init(&bar_dq, 1);
    fence_barrier_init();
  }
  if (warp == ISSUER_WARP) tmem_alloc(&tmem_base_s, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_base_s;      // S: [0,128), g_P: [128,256), g_q: [256, 256 + D)
  pdl_wait();
  pdl_launch_dependents();
  const uint32_t sb = smem_u32(smem);

  if (warp == ISSUER_WARP) {
    // ---------------------------------------------------------------- TMA + MMA issue
    constexpr uint64_t dk = smem_desc_sw128(16, 1024), dmn = smem_desc_sw128(CH, 1024);
    constexpr uint32_t idesc_s = idesc_bf16(BQ, BKEY, 0, 0), idesc_q = idesc_bf16(BQ, D, 0, 1);
    // the K / V tiles of the 2 nkb iterations (two sweeps) go round NKV buffers
    auto load_kv = [&](int it) {
      const int b = it % B::NKV, kb = it % nkb;
      if (elect_one_sync()) {
        mbar_expect_tx(&bar_kv[b], B::PAIR);
        for (int c = 0; c < B::NC; ++c) {
          tma_load_3d(smem + B::KV_OFF + b * B::PAIR + c * CH, &mapQ, &bar_kv[b], p.C + h * D + 64 * c, kb * BKEY, n);
          tma_load_3d(smem + B::KV_OFF + b * B::PAIR + B::NC * CH + c * CH, &mapQ, &bar_kv[b], 2 * p.C + h * D + 64 * c, kb * BKEY, n);
        }
      }
    };
    auto issue_dq = [&](int j) {            // j: key tile of sweep 2; its K tile is the one of iteration nkb + j
      mbar_wait(&bar_ds, j & 1);
      tc_fence_after();
      const uint32_t kt = sb + B::KV_OFF + ((nkb + j) % B::NKV) * B::PAIR;
#pragma unroll
      for (int k = 0; k < BKEY / 16; ++k)
        if (elect_one_sync())
          umma_bf16(tmem + 256, desc_with_addr(dk, sb + B::DS_OFF + (k / 4) * CH + (k % 4) * 32), desc_with_addr(dmn, kt + k * 2048),
                    idesc_q, (j | k) != 0);
      if (elect_one_sync()) umma_commit(&bar_dq);
      __syncwarp();
    };
    if (elect_one_sync()) {
      mbar_expect_tx(&bar_q, 2 * B::NC * CH);
      for (int c = 0; c < B::NC; ++c) {
        tma_load_3d(smem + B::Q_OFF + c * CH, &mapQ, &bar_q, h * D + 64 * c, q0, n);
        tma_load_3d(smem + B::GO_OFF + c * CH, &mapG, &bar_q, h * D + 64 * c, q0, n);
      }
    }
    load_kv(0);
    mbar_wait(&bar_q, 0);
    for (int it = 0; it < nit; ++it) {
      const int b = it % B::NKV;
      mbar_wait(&bar_kv[b], (it / B::NKV) & 1);
      if (it > 0) mbar_wait(&bar_sfree, (it - 1) & 1);
      tc_fence_after();
      const uint32_t kv = sb + B::KV_OFF + b * B::PAIR;
#pragma unroll
      for (int k = 0; k < D / 16; ++k) {      // S = Q K^T
        const uint32_t off = (k / 4) * CH + (k % 4) * 32;
        if (elect_one_sync()) umma_bf16(tmem, desc_with_addr(dk, sb + B::Q_OFF + off), desc_with_addr(dk, kv + off), idesc_s, k != 0);
      }
#pragma unroll
      for (int k = 0; k < D / 16; ++k) {      // g_P = g_o V^T
        const uint32_t off = (k / 4) * CH + (k % 4) * 32;
        if (elect_one_sync())
          umma_bf16(tmem + 128, desc_with_addr(dk, sb + B::GO_OFF + off), desc_with_addr(dk, kv + B::NC * CH + off), idesc_s, k != 0);
      }
      if (elect_one_sync()) umma_commit(&bar_s);
      __syncwarp();
      // The tile of iteration it + 1 goes into the buffer that iteration it + 1 - NKV used.  Its S / g_P are complete
      // (bar_sfree); in sweep 2 its g_S K must be, too.  Three buffers (d = 64): that is the product of iteration it - 2,
      // issued one iteration ago, and it is waited for BEFORE the next one is issued (bar_dq must not run two phases ahead
      // of a parity wait).  Two buffers (d = 128): the product issued in this iteration.
      if (B::NKV == 3) {
        if (it - 2 >= nkb) mbar_wait(&bar_dq, (it - 2 - nkb) & 1);
        if (it + 1 < nit) load_kv(it + 1);
      }
      if (it > nkb) issue_dq(it - 1 - nkb);
      if (B::NKV == 2) {
        if (it - 1 >= nkb) mbar_wait(&bar_dq, (it - 1 - nkb) & 1);
        if (it + 1 < nit) load_kv(it + 1);
      }
    }
    issue_dq(nkb - 1);
  } else {
    // ---------------------------------------------------------------- softmax threads: (query row, half of the key columns)
    const int row = threadIdx.x & (BQ - 1), half = threadIdx.x >> 7;
    const uint32_t trow = tmem + ((uint32_t)((warp & 3) * 32) << 16);
    const int q = q0 + row;
    const float c2 = p.scale * 1.4426950408889634f;
    const float lse2 = (q < p.T ? p.lse[((size_t)n * p.heads + h) * p.T + q] : 0.f) * 1.4426950408889634f;
    const f2_t c22 = pk2(c2, c2), ml2 = pk2(-lse2, -lse2);
    float Dr = 0.f;
    f2_t D2 = pk2(0.f, 0.f), mD2 = D2;
    for (int it = 0; it < nit; ++it) {
      const int kb = it % nkb;
      if (it == nkb) {                     // between the sweeps: D_i of the two column halves
        float t0, t1;
        upk2(D2, t0, t1);
        xch[half][row] = Dr + t0 + t1;
        softmax_sync();
        Dr = xch[0][row] + xch[1][row];
        if (q < p.T && half == 0) p.Dg[((size_t)n * p.heads + h) * p.T + q] = Dr;
        mD2 = pk2(-Dr, -Dr);
      }
      mbar_wait(&bar_s, it & 1);
      tc_fence_after();
      uint32_t rs0[32], rs1[32], rp0[32], rp1[32];
      tmem_ld32(trow + (2 * half) * 32, rs0);
      tmem_ld32(trow + (2 * half + 1) * 32, rs1);
      tmem_ld32(trow + 128 + (2 * half) * 32, rp0);
      tmem_ld32(trow + 128 + (2 * half + 1) * 32, rp1);
      tmem_ld_wait();
      tc_fence_before();
      mbar_arrive(&bar_sfree);
      const int kbase = kb * BKEY + 2 * half * 32;
      const bool ragged = (kb + 1) * BKEY > p.T;
      if (it < nkb) {
        // ---- sweep 1: D_i = sum_j P_ij g_P_ij
        if (!ragged) {
#pragma unroll
          for (int i = 0; i < 32; i += 2) {
            float a0, a1;
            upk2(fma2(pk2(__uint_as_float(rs0[i]), __uint_as_float(rs0[i + 1])), c22, ml2), a0, a1);
            D2 = fma2(pk2(ex2a(a0), ex2a(a1)), pk2(__uint_as_float(rp0[i]), __uint_as_float(rp0[i + 1])), D2);
            upk2(fma2(pk2(__uint_as_float(rs1[i]), __uint_as_float(rs1[i + 1])), c22, ml2), a0, a1);
            D2 = fma2(pk2(ex2a(a0), ex2a(a1)), pk2(__uint_as_float(rp1[i]), __uint_as_float(rp1[i + 1])), D2);
          }
        } else {
#pragma unroll
          for (int i = 0; i < 32; ++i) {
            if (kbase + i < p.T) Dr = fmaf(ex2a(fmaf(__uint_as_float(rs0[i]), c2, -lse2)), __uint_as_float(rp0[i]), Dr);
            if (kbase + 32 + i < p.T) Dr = fmaf(ex2a(fmaf(__uint_as_float(rs1[i]), c2, -lse2)), __uint_as_float(rp1[i]), Dr);
          }
        }
        continue;
      }
      // ---- sweep 2: g_S = P (g_P - D) as bf16 into the A tile
      uint32_t pk0[16], pk1[16];
      if (!ragged) {
#pragma unroll
        for (int i = 0; i < 32; i += 2) {
          float a0, a1, d0, d1;
          upk2(fma2(pk2(__uint_as_float(rs0[i]), __uint_as_float(rs0[i + 1])), c22, ml2), a0, a1);
          upk2(mul2(pk2(ex2a(a0), ex2a(a1)), add2(pk2(__uint_as_float(rp0[i]), __uint_as_float(rp0[i + 1])), mD2)), d0, d1);
          pk0[i >> 1] = pack_bf16(d0, d1);
          upk2(fma2(pk2(__uint_as_float(rs1[i]), __uint_as_float(rs1[i + 1])), c22, ml2), a0, a1);
          upk2(mul2(pk2(ex2a(a0), ex2a(a1)), add2(pk2(__uint_as_float(rp1[i]), __uint_as_float(rp1[i + 1])), mD2)), d0, d1);
          pk1[i >> 1] = pack_bf16(d0, d1);
        }
      } else {
#pragma unroll
        for (int i = 0; i < 32; i += 2) {
          float d0 = kbase + i < p.T ? ex2a(fmaf(__uint_as_float(rs0[i]), c2, -lse2)) * (__uint_as_float(rp0[i]) - Dr) : 0.f;
          float d1 = kbase + i + 1 < p.T ? ex2a(fmaf(__uint_as_float(rs0[i + 1]), c2, -lse2)) * (__uint_as_float(rp0[i + 1]) - Dr) : 0.f;
          pk0[i >> 1] = pack_bf16(d0, d1);
          d0 = kbase + 32 + i < p.T ? ex2a(fmaf(__uint_as_float(rs1[i]), c2, -lse2)) * (__uint_as_float(rp1[i]) - Dr) : 0.f;
          d1 = kbase + 32 + i + 1 < p.T ? ex2a(fmaf(__uint_as_float(rs1[i + 1]), c2, -lse2)) * (__uint_as_float(rp1[i + 1]) - Dr) : 0.f;
          pk1[i >> 1] = pack_bf16(d0, d1);
        }
      }
      if (it > nkb) mbar_wait(&bar_dq, (it - 1 - nkb) & 1);      // the previous g_S K has read g_S
      store_row_chunk32(sb + B::DS_OFF, row, 2 * half, pk0);
      store_row_chunk32(sb + B::DS_OFF, row, 2 * half + 1, pk1);
      fence_proxy_async_smem();
      mbar_arrive(&bar_ds);
    }
    mbar_wait(&bar_dq, (nkb - 1) & 1);
    tc_fence_after();
    bf16* gq = p.g_qkv + ((size_t)n * p.T + q) * 3 * p.C + (size_t)h * D;
#pragma unroll
    for (int cc = 0; cc < D / 64; ++cc) {
      const int ch = half * (D / 64) + cc;
      uint32_t r[32];
      tmem_ld32(trow + 256 + ch * 32, r);
      tmem_ld_wait();
      if (q < p.T) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          uint4 v;
          v.x = pack_bf16(__uint_as_float(r[8 * j]) * p.scale, __uint_as_float(r[8 * j + 1]) * p.scale);
          v.y = pack_bf16(__uint_as_float(r[8 * j + 2]) * p.scale, __uint_as_float(r[8 * j + 3]) * p.scale);
          v.z = pack_bf16(__uint_as_float(r[8 * j + 4]) * p.scale, __uint_as_float(r[8 * j + 5]) * p.scale);
          v.w = pack_bf16(__uint_as_float(r[8 * j + 6]) * p.scale, __uint_as_float(r[8 * j + 7]) * p.scale);
          *reinterpret_cast<uint4*>(gq + ch * 32 + 8 * j) = v;
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == ISSUER_WARP) {
    tc_fence_after();
    tmem_dealloc(tmem, 512);
  }
}

template <int D>
__global__ void __launch_bounds__(FWD_THREADS, 1) attn_bwd_dkv_tc_k(const __grid_constant__ CUtensorMap mapQ,
                                                                    const __grid_constant__ CUtensorMap mapG, const AtbP p) {
  using B = BCfg<D>;
  extern __shared__ uint8_t smem_raw[];
  // bar_s: S and g_P complete | bar_sfree: both are in registers | bar_p: P and g_S written | bar_acc: g_v += P^T g_o and
  // g_k += g_S^T Q complete (P, g_S and that Q / g_o tile are free)
  __shared__ uint64_t bar_kv, bar_q[B::NQB], bar_s, bar_sfree, bar_p, bar_acc;
  __shared__ uint32_t tmem_base_s;
  uint8_t* smem = smem_raw + ((1024 - (smem_u32(smem_raw) & 1023)) & 1023);
  const int warp = threadIdx.x >> 5;
  const int k0 = blockIdx.x * BKEY, h = blockIdx.y, n = blockIdx.z;
  const int nqb = (p.T + BQ - 1) / BQ;
  if (threadIdx.x == 0) {
    prefetch_tmap(&mapQ); prefetch_tmap(&mapG);
    mbar_init(&bar_kv, 1);
    for (int b = 0; b < B::NQB; ++b) mbar_init(&bar_q[b], 1);
    mbar_init(&bar_s, 1); mbar_init(&bar_sfree, SOFTMAX_THREADS); mbar_init(&bar_p, SOFTMAX_THREADS); mbar_init(&bar_acc, 1);
    fence_barrier_init();
  }
  if (warp == ISSUER_WARP) tmem_alloc(&tmem_base_s, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_base_s;      // S: [0,128), g_P: [128,256), g_v: [256, 256 + D), g_k: [256 + D, 256 + 2 D)
  pdl_wait();
  pdl_launch_dependents();
  const uint32_t sb = smem_u32(smem);

  if (warp == ISSUER_WARP) {
    // ---------------------------------------------------------------- TMA + MMA issue
    constexpr uint64_t dk = smem_desc_sw128(16, 1024), dmn = smem_desc_sw128(CH, 1024);
    constexpr uint32_t idesc_s = idesc_bf16(BQ, BKEY, 0, 0), idesc_t = idesc_bf16(BKEY, D, 1, 1);
    if (elect_one_sync()) {                 // this CTA's keys: K, V resident
      mbar_expect_tx(&bar_kv, 2 * B::NC * CH);
      for (int c = 0; c < B::NC; ++c) {
        tma_load_3d(smem + B::K_OFF + c * CH, &mapQ, &bar_kv, p.C + h * D + 64 * c, k0, n);
        tma_load_3d(smem + B::V_OFF + c * CH, &mapQ, &bar_kv, 2 * p.C + h * D + 64 * c, k0, n);
      }
    }
    auto load_q = [&](int qb) {             // Q and g_o of a query block
      const int b = qb % B::NQB;
      if (elect_one_sync()) {
        mbar_expect_tx(&bar_q[b], B::PAIR);
        for (int c = 0; c < B::NC; ++c) {
          tma_load_3d(smem + B::QG_OFF + b * B::PAIR + c * CH, &mapQ, &bar_q[b], h * D + 64 * c, qb * BQ, n);
          tma_load_3d(smem + B::QG_OFF + b * B::PAIR + B::NC * CH + c * CH, &mapG, &bar_q[b], h * D + 64 * c, qb * BQ, n);
        }
      }
    };
    auto issue_acc = [&](int j) {           // g_v += P^T g_o, g_k += g_S^T Q of query block j
      mbar_wait(&bar_p, j & 1);
      tc_fence_after();
      const uint32_t qg = sb + B::QG_OFF + (j % B::NQB) * B::PAIR;
      // A = P^T / g_S^T: the [query][key] tiles read MN-major (M = keys: two 64-key chunks, LBO = CH; K = 16 query rows per step)
#pragma unroll
      for (int k = 0; k < BQ / 16; ++k)
        if (elect_one_sync())
          umma_bf16(tmem + 256, desc_with_addr(dmn, sb + B::P_OFF + k * 2048), desc_with_addr(dmn, qg + B::NC * CH + k * 2048),
                    idesc_t, (j | k) != 0);
#pragma unroll
      for (int k = 0; k < BQ / 16; ++k)
        if (elect_one_sync())
          umma_bf16(tmem + 256 + D, desc_with_addr(dmn, sb + B::DS2_OFF + k * 2048), desc_with_addr(dmn, qg + k * 2048),
                    idesc_t, (j | k) != 0);
      if (elect_one_sync()) umma_commit(&bar_acc);
      __syncwarp();
    };
    if (B::NQB == 3) load_q(0);
    mbar_wait(&bar_kv, 0);
    for (int qb = 0; qb < nqb; ++qb) {
      const int b = qb % B::NQB;
      if (B::NQB == 1) {                    // one Q / g_o buffer (d = 128): the previous block's products first
        if (qb > 0) { issue_acc(qb - 1); mbar_wait(&bar_acc, (qb - 1) & 1); }
        load_q(qb);
      }
      mbar_wait(&bar_q[b], (qb / B::NQB) & 1);
      if (qb > 0) mbar_wait(&bar_sfree, (qb - 1) & 1);
      tc_fence_after();
      const uint32_t qg = sb + B::QG_OFF + b * B::PAIR;
#pragma unroll
      for (int k = 0; k < D / 16; ++k) {
        const uint32_t off = (k / 4) * CH + (k % 4) * 32;
        if (elect_one_sync()) umma_bf16(tmem, desc_with_addr(dk, qg + off), desc_with_addr(dk, sb + B::K_OFF + off), idesc_s, k != 0);
      }
#pragma unroll
      for (int k = 0; k < D / 16; ++k) {
        const uint32_t off = (k / 4) * CH + (k % 4) * 32;
        if (elect_one_sync())
          umma_bf16(tmem + 128, desc_with_addr(dk, qg + B::NC * CH + off), desc_with_addr(dk, sb + B::V_OFF + off), idesc_s, k != 0);
      }
      if (elect_one_sync()) umma_commit(&bar_s);
      __syncwarp();
      if (B::NQB == 3) {
        // block qb + 1 goes into the buffer block qb - 2 used: its products (issued one iteration ago) are waited for
        // BEFORE the next ones are issued (bar_acc must not run two phases ahead of a parity wait)
        if (qb >= 2) mbar_wait(&bar_acc, (qb - 2) & 1);
        if (qb + 1 < nqb) load_q(qb + 1);
        if (qb > 0) issue_acc(qb - 1);
      }
    }
    issue_acc(nqb - 1);
  } else {
    // ---------------------------------------------------------------- softmax threads: (query row, half of this CTA's keys)
    const int row = threadIdx.x & (BQ - 1), half = threadIdx.x >> 7;
    const uint32_t trow = tmem + ((uint32_t)((warp & 3) * 32) << 16);
    const float c2 = p.scale * 1.4426950408889634f;
    const f2_t c22 = pk2(c2, c2);
    for (int qb = 0; qb < nqb; ++qb) {
      const int q = qb * BQ + row;
      // rows past the end: Q and g_o are zero-filled by TMA, so with lse = D = 0 their P = 1 and g_S = 0 meet zero rows of
      // g_o / Q in the products: no masks
      const float lse2 = (q < p.T ? p.lse[((size_t)n * p.heads + h) * p.T + q] : 0.f) * 1.4426950408889634f;
      const float Dr = q < p.T ? p.Dg[((size_t)n * p.heads + h) * p.T + q] : 0.f;
      const f2_t ml2 = pk2(-lse2, -lse2), mD2 = pk2(-Dr, -Dr);
      mbar_wait(&bar_s, qb & 1);
      tc_fence_after();
      uint32_t rs0[32], rs1[32], rp0[32], rp1[32];
      tmem_ld32(trow + (2 * half) * 32, rs0);
      tmem_ld32(trow + (2 * half + 1) * 32, rs1);
      tmem_ld32(trow + 128 + (2 * half) * 32, rp0);
      tmem_ld32(trow + 128 + (2 * half + 1) * 32, rp1);
      tmem_ld_wait();
      tc_fence_before();
      mbar_arrive(&bar_sfree);
      uint32_t pp0[16], pp1[16], pd0[16], pd1[16];
#pragma unroll
      for (int i = 0; i < 32; i += 2) {
        float a0, a1, d0, d1;
        upk2(fma2(pk2(__uint_as_float(rs0[i]), __uint_as_float(rs0[i + 1])), c22, ml2), a0, a1);
        a0 = ex2a(a0); a1 = ex2a(a1);
        pp0[i >> 1] = pack_bf16(a0, a1);
        upk2(mul2(pk2(a0, a1), add2(pk2(__uint_as_float(rp0[i]), __uint_as_float(rp0[i + 1])), mD2)), d0, d1);
        pd0[i >> 1] = pack_bf16(d0, d1);
        upk2(fma2(pk2(__uint_as_float(rs1[i]), __uint_as_float(rs1[i + 1])), c22, ml2), a0, a1);
        a0 = ex2a(a0); a1 = ex2a(a1);
        pp1[i >> 1] = pack_bf16(a0, a1);
        upk2(mul2(pk2(a0, a1), add2(pk2(__uint_as_float(rp1[i]), __uint_as_float(rp1[i + 1])), mD2)), d0, d1);
        pd1[i >> 1] = pack_bf16(d0, d1);
      }
      if (qb > 0) mbar_wait(&bar_acc, (qb - 1) & 1);      // the previous products have read P and g_S
      store_row_chunk32(sb + B::P_OFF, row, 2 * half, pp0);
      store_row_chunk32(sb + B::P_OFF, row, 2 * half + 1, pp1);
      store_row_chunk32(sb + B::DS2_OFF, row, 2 * half, pd0);
      store_row_chunk32(sb + B::DS2_OFF, row, 2 * half + 1, pd1);
      fence_proxy_async_smem();
      mbar_arrive(&bar_p);
    }
    mbar_wait(&bar_acc, (nqb - 1) & 1);
    tc_fence_after();
    const int key = k0 + row;
    bf16* gk = p.g_qkv + ((size_t)n * p.T + key) * 3 * p.C + (size_t)h * D + p.C;
#pragma unroll
    for (int part = 0; part < 2; ++part) {       // 0: g_v (unscaled) -> third 2; 1: g_k (x scale) -> third 1
      const float f = part ? p.scale : 1.0f;
      bf16* dst = part ? gk : gk + p.C;
#pragma unroll
      for (int cc = 0; cc < D / 64; ++cc) {
        const int ch = half * (D / 64) + cc;
        uint32_t r[32];
        tmem_ld32(trow + 256 + part * D + ch * 32, r);
        tmem_ld_wait();
        if (key < p.T) {
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            uint4 v;
            v.x = pack_bf16(__uint_as_float(r[8 * j]) * f, __uint_as_float(r[8 * j + 1]) * f);
            v.y = pack_bf16(__uint_as_float(r[8 * j + 2]) * f, __uint_as_float(r[8 * j + 3]) * f);
            v.z = pack_bf16(__uint_as_float(r[8 * j + 4]) * f, __uint_as_float(r[8 * j + 5]) * f);
            v.w = pack_bf16(__uint_as_float(r[8 * j + 6]) * f, __uint_as_float(r[8 * j + 7]) * f);
            *reinterpret_cast<uint4*>(dst + ch * 32 + 8 * j) = v;
          }
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == ISSUER_WARP) {
    tc_fence_after();
    tmem_dealloc(tmem, 512);
  }
}

template <int D> bool launch_atb(const CUtensorMap& mq, const CUtensorMap& mg, const AtbP& p, int n, cudaStream_t st) {
  static bool attr = false;
  if (!attr) {
    if (cudaFuncSetAttribute(attn_bwd_dq_tc_k<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, BCfg<D>::SMEM_DQ) != cudaSuccess ||
        cudaFuncSetAttribute(attn_bwd_dkv_tc_k<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, BCfg<D>::SMEM_DKV) != cudaSuccess)
      return false;
    attr = true;
  }
  const dim3 grid((p.T + BQ - 1) / BQ, p.heads, n);
  // the second kernel reads D, which the first one writes after its dependency wait: ordinary stream order between the two
  if (launch_pdl(attn_bwd_dq_tc_k<D>, grid, dim3(FWD_THREADS), BCfg<D>::SMEM_DQ, st, mq, mg, p) != cudaSuccess) return false;
  return launch_pdl(attn_bwd_dkv_tc_k<D>, grid, dim3(FWD_THREADS), BCfg<D>::SMEM_DKV, st, mq, mg, p) == cudaSuccess;
}

template <int D> bool launch_atc(const CUtensorMap& map, const AtcP& p, int n, cudaStream_t st) {
  static bool attr = false;
  if (!attr) {
    if (cudaFuncSetAttribute(attn_fwd_tc_k<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, ACfg<D>::SMEM) != cudaSuccess) return false;
    attr = true;
  }
  return launch_pdl(attn_fwd_tc_k<D>, dim3((p.T + BQ - 1) / BQ, p.heads, n), dim3(FWD_THREADS), ACfg<D>::SMEM, st, map, p) == cudaSuccess;
}

}  // namespace

bool attn_fwd_tc_supported(int dt, int C, int heads) {
  if (dt != DT_BF16 || heads <= 0 || C % heads) return false;
  const int d = C / heads;
  return d == 64 || d == 128;
}

// 1 on launch, -1 on failure (tensor map / attribute)
int attn_fwd_tc(const void* qkv, int n, int T, int C, int heads, void* o, float* lse, cudaStream_t st) {
  CUtensorMap map;
  const uint64_t dims[3] = {(uint64_t)3 * C, (uint64_t)T, (uint64_t)n};
  const uint64_t str[2] = {(uint64_t)3 * C * 2, (uint64_t)T * 3 * C * 2};
  const uint32_t box[3] = {64, BQ, 1};
  if (!tmap::get_map(qkv, 3, dims, str, box, &map)) return -1;
  AtcP p;
  p.T = T; p.C = C; p.heads = heads; p.scale = 1.0f / sqrtf((float)(C / heads)); p.o = (bf16*)o; p.lse = lse;
  const bool ok = C / heads == 64 ? launch_atc<64>(map, p, n, st) : launch_atc<128>(map, p, n, st);
  return ok ? 1 : -1;
}

// 2 on launch, -1 on failure.  stats: [log-sum-exp | D] as attn_stats_floats lays them out
int attn_bwd_tc(const void* qkv, const void* g_o, int n, int T, int C, int heads, float* stats, void* g_qkv, cudaStream_t st) {
  CUtensorMap mq, mg;
  const uint32_t box[3] = {64, BQ, 1};
  {
    const uint64_t dims[3] = {(uint64_t)3 * C, (uint64_t)T, (uint64_t)n};
    const uint64_t str[2] = {(uint64_t)3 * C * 2, (uint64_t)T * 3 * C * 2};
    if (!tmap::get_map(qkv, 3, dims, str, box, &mq)) return -1;
  }
  {
    const uint64_t dims[3] = {(uint64_t)C, (uint64_t)T, (uint64_t)n};
    const uint64_t str[2] = {(uint64_t)C * 2, (uint64_t)T * C * 2};
    if (!tmap::get_map(g_o, 3, dims, str, box, &mg)) return -1;
  }
  AtbP p;
  p.T = T; p.C = C; p.heads = heads; p.scale = 1.0f / sqrtf((float)(C / heads)); p.g_qkv = (bf16*)g_qkv;
  p.lse = stats; p.Dg = stats + (size_t)n * heads * T;
  const bool ok = C / heads == 64 ? launch_atb<64>(mq, mg, p, n, st) : launch_atb<128>(mq, mg, p, n, st);
  return ok ? 2 : -1;
}

}  // namespace pulse

// conv_tc2.cu - CTA-pair (tcgen05 cta_group::2) implicit-GEMM convolution for sm_100a.
//
// Same GEMM view as conv_tc.cu (D[pixel, co] = sum_{tap, c} A[pixel shifted by tap, c] W[co][tap][c], TMA im2col
// by coordinate shift with hardware zero fill, virtual concat by switching tensor maps inside the K loop), but the
// tile is computed by TWO CTAs of a cluster on neighbouring SMs:
//   pair tile   = 256 pixels x (NJ x UN) output channels; each CTA owns 128 of the pixels (its TMEM lanes),
//   per K block = each CTA loads ITS 128 pixel rows of A and HALF of the weight rows of every UN-wide N slice;
//                 one thread of the leader CTA issues tcgen05.mma.cta_group::2 (M = 256, N = UN), which reads A and
//                 B from both CTAs' shared memory and accumulates into both CTAs' TMEM.
// Why: the 128 x 160 single-CTA tile fetches 36.9 KB of operands per 2.6 MFLOP (71 FLOP/B) and its main loop is
// bound by that operand feed (profiles/r01a_*: tensor pipe 51 % active).  The 256 x 320 pair tile fetches the same
// 36.9 KB per CTA for twice the math (142 FLOP/B) and halves each CTA's shared-memory read traffic per MMA.
//
// Synchronisation (barriers live at the same shared-memory offsets in both CTAs):
//   full[s]   (leader's copy)  1 arrival: the leader's producer arrive.expect_tx(bytes of BOTH CTAs); the TMA loads
//                              of both CTAs complete_tx on it (cp.async.bulk.tensor ... cta_group::2),
//   empty[s]  (own copy)       tcgen05.commit multicast to both CTAs when the MMAs reading stage s are done,
//   tfull[a]  (own copy)       tcgen05.commit multicast when a tile's accumulator is complete,
//   tempty[a] (leader's copy)  8 arrivals: the 4 epilogue warps of both CTAs (remote arrive from the peer).
//
// Split-K over a cluster (SK = 2 or 4 pairs, cluster of 2 SK CTAs) for convs with few tiles and a long K (1280 channels on
// 8x8 / 16x16 pixels: 8 / 32 pair tiles for 74 pairs): the SK pairs of a cluster take the SAME output tile and 1/SK of the
// K blocks each.  The partial accumulators meet through distributed shared memory: the tile's 32-channel chunks are dealt
// round-robin to the SK pairs; every CTA writes the chunks it does not own into the owner's (by then idle) operand ring
// (st.shared::cluster, 16 KB per chunk and sender), the owner adds them to its TMEM chunk and runs the ordinary epilogue on
// it.  Two cluster barriers: all rings idle / all partials delivered.  One tile per cluster.
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

constexpr int BM = 128, BK = 64;
constexpr int A_BYTES = BM * BK * 2;           // 16 KB

// A launch covers 1 or 4 PHASES (stride-2 dgrad, 4-phase upsample conv): sub-pixel convs that share the source, the
// pixel grid and the weight matrix's K layout but have their own taps, weight rows and output parity.  Phases are extra
// tiles of one persistent launch, so small grids still fill the machine.
struct Tc2Params {
  int c0_blocks, c_blocks, ctot, c0;
  int s2;                         // 1: stride-2 fprop through the 5-D parity view
  int nph, ph_tap0[5], ph_wrow[4], ph_ooy[4], ph_oox[4];      // phase i: taps [ph_tap0[i], ph_tap0[i+1]), first weight row, output parity
  Tap taps[16];
  int bw, bh, bn, tiles_h, tiles_m, pair_tiles_m, n_tiles;
  int GH, GN;                     // pixel grid (rows, images); columns == bw
  const bf16* bias; const float* pn; const bf16* residual; bf16* out; int accumulate;
  int OH, OW, osy, osx, cout_total;
  float* cst;                     // channel stats [n][2][cout] of the stored output, accumulated (or null)
};
// one output view per phase; MP = false: the one-phase launch's kernel carries one map (0.5 KB less of kernel parameters)
template <bool MP> struct OutMaps { CUtensorMap m[MP ? 4 : 1]; };

template <int UN, int NJ> struct Cfg2 {
  static constexpr int BN = UN * NJ;                       // output channels per pair tile
  static constexpr int B_SLICE = (UN / 2) * BK * 2;        // this CTA's half of one UN-wide weight slice
  static constexpr int STAGE_BYTES = A_BYTES + NJ * B_SLICE;
  static constexpr int CW = 32;                            // channels per epilogue chunk / TMA store box
  static constexpr int BOX_BYTES = 32 * CW * 2;            // one warp's [32 pixels][CW channels] bf16
  static constexpr int NBUF = 2;                           // staging boxes per warp: chunk c is written while the TMA store of c - 1 reads
  static constexpr int EPI_BYTES = 4 * (2 * NBUF * BOX_BYTES + 2048);   // per quadrant: 2 warps x NBUF boxes + column vector [BN] fp32
  static constexpr int RING = 227 * 1024 - 256 - EPI_BYTES - 1024;       // what is left of the 227 KB for the operand ring
  static constexpr int STAGES = RING / STAGE_BYTES > 8 ? 8 : RING / STAGE_BYTES;
  static constexpr int SMEM = STAGES * STAGE_BYTES + EPI_BYTES + 1024;
  static constexpr int ACC = 2 * BN <= 512 ? 2 : 1;        // TMEM accumulator stages
  static constexpr int TMEM_COLS = ACC * BN <= 256 ? 256 : 512;
  static_assert(B_SLICE % 1024 == 0, "weight slices must keep the 1024-byte swizzle-atom alignment");
  static_assert(UN % 16 == 0 && UN <= 256, "UMMA N for M = 256");
};

template <int UN, int NJ, bool MP, int SK>
__global__ void __cluster_dims__(2 * SK, 1, 1) __launch_bounds__(320, 1)
conv_tc2_k(const __grid_constant__ CUtensorMap mapA0, const __grid_constant__ CUtensorMap mapA1,
           const __grid_constant__ CUtensorMap mapB, const __grid_constant__ OutMaps<MP> mapO, const Tc2Params p) {
  using C = Cfg2<UN, NJ>;
  extern __shared__ uint8_t smem_raw[];
  __shared__ uint64_t full_bar[C::STAGES], empty_bar[C::STAGES], tfull_bar[2], tempty_bar[2];
  __shared__ uint32_t tmem_base_s;
  uint8_t* smem = smem_raw + ((1024 - (smem_u32(smem_raw) & 1023)) & 1023);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // rank: this CTA inside its pair; lead: cluster rank of the pair's leader; ks: which share of the K blocks (split-K)
  const uint32_t crank = cluster_ctarank();
  const uint32_t rank = SK == 1 ? crank : (crank & 1u), lead = SK == 1 ? 0u : (crank & ~1u);
  const int ks = SK == 1 ? 0 : (int)(crank >> 1);
  const uint16_t pair_mask = (uint16_t)(3u << lead);
  const int tiles_ph = p.pair_tiles_m * p.n_tiles;      // tiles per phase
  const int total_tiles = p.nph * tiles_ph;
  const int pair = blockIdx.x / (2 * SK), npairs = gridDim.x / (2 * SK);      // tile walkers: pairs, or clusters of SK pairs

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&mapA0); prefetch_tmap(&mapA1); prefetch_tmap(&mapB); prefetch_tmap(&mapO.m[0]);
    for (int i = 0; i < C::STAGES; ++i) { mbar_init(&full_bar[i], 1); mbar_init(&empty_bar[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&tfull_bar[i], 1); mbar_init(&tempty_bar[i], 16); }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc2(&tmem_base_s, C::TMEM_COLS);
  tc_fence_before();
  cluster_sync_all();          // the peer's barriers are initialised and its TMEM allocated before anyone signals
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_s;
  pdl_wait();                  // everything above overlapped the tail of the previous kernel
  pdl_launch_dependents();

  if (warp == 0) {
    if (lane == 0) {
      // ===== TMA producer (both CTAs): own 128 pixel rows of A, own half of every weight slice =====
      int stage = 0; uint32_t phase = 0;
      for (int tile = pair; tile < total_tiles; tile += npairs) {
        const int ph = tile / tiles_ph, tl = tile - ph * tiles_ph;
        const int mp = tl / p.n_tiles, nt = tl - mp * p.n_tiles;
        const int mt = 2 * mp + (int)rank;
        const int n0 = (mt / p.tiles_h) * p.bn, y0 = (mt % p.tiles_h) * p.bh;
        const int tap0 = p.ph_tap0[ph], num_kb = (p.ph_tap0[ph + 1] - tap0) * p.c_blocks, wrow = p.ph_wrow[ph];
        const int kb0 = SK == 1 ? 0 : ks * num_kb / SK, kb1 = SK == 1 ? num_kb : (ks + 1) * num_kb / SK;
        for (int kb = kb0; kb < kb1; ++kb) {
          const int ti = kb / p.c_blocks, cb = kb - ti * p.c_blocks;
          const Tap t = p.taps[tap0 + ti];
          mbar_wait(&empty_bar[stage], phase ^ 1);
          if (rank == 0) mbar_expect_tx(&full_bar[stage], 2 * C::STAGE_BYTES);
          const uint32_t fb = mapa_u32(smem_u32(&full_bar[stage]), lead);
          uint8_t* sa = smem + stage * C::STAGE_BYTES;
          const bool first = cb < p.c0_blocks;
          const CUtensorMap* ma = first ? &mapA0 : &mapA1;
          const int cch = (first ? cb : cb - p.c0_blocks) * BK;
          if (!p.s2) tma2_load_4d(sa, ma, fb, cch, t.dx, y0 + t.dy, n0);
          else tma2_load_5d(sa, ma, fb, t.px * p.c0 + cch, t.dx, t.py, y0 + t.dy, n0);
          const int kcol = t.widx * p.ctot + cb * BK;
#pragma unroll
          for (int j = 0; j < NJ; ++j)
            tma2_load_2d(sa + A_BYTES + j * C::B_SLICE, &mapB, fb, kcol, wrow + nt * C::BN + j * UN + (int)rank * (UN / 2));
          if (++stage == C::STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    if (rank == 0) {
      // ===== MMA issuer (leader CTA only): the whole warp runs the loop, one elected lane issues =====
      constexpr uint32_t idesc = idesc_bf16(2 * BM, UN, 0, 0);
      constexpr uint64_t dbase = smem_desc_sw128(16, 1024);
      constexpr uint32_t desc_hi = (uint32_t)(dbase >> 32);
      const uint32_t desc_lo0 = (uint32_t)dbase | ((smem_u32(smem) >> 4) & 0x3FFF);     // smem is 1024-aligned: no carry
      int stage = 0; uint32_t phase = 0; int acc = 0; uint32_t acc_phase = 0;
      for (int tile = pair; tile < total_tiles; tile += npairs) {
        const int ph = tile / tiles_ph;
        const int num_kb = (p.ph_tap0[ph + 1] - p.ph_tap0[ph]) * p.c_blocks;
        mbar_wait(&tempty_bar[acc], acc_phase ^ 1);
        tc_fence_after();
        const uint32_t tmem_d = tmem_base + acc * C::BN;
        const int kb0 = SK == 1 ? 0 : ks * num_kb / SK, kb1 = SK == 1 ? num_kb : (ks + 1) * num_kb / SK;
        for (int kb = kb0; kb < kb1; ++kb) {
          mbar_wait(&full_bar[stage], phase);
          tc_fence_after();
          const uint32_t a_lo = desc_lo0 + stage * (C::STAGE_BYTES >> 4), b_lo = a_lo + (A_BYTES >> 4);
          if (elect_one_sync()) {
#pragma unroll
            for (int k = 0; k < BK / 16; ++k)
#pragma unroll
              for (int j = 0; j < NJ; ++j)
                umma2_bf16(tmem_d + j * UN, ((uint64_t)desc_hi << 32) | (a_lo + 2 * k),
                           ((uint64_t)desc_hi << 32) | (b_lo + j * (C::B_SLICE >> 4) + 2 * k), idesc, ((kb - kb0) | k) != 0);
            umma2_commit_mc(&empty_bar[stage], pair_mask);
            if (kb == kb1 - 1) umma2_commit_mc(&tfull_bar[acc], pair_mask);
          }
          __syncwarp();
          if (++stage == C::STAGES) { stage = 0; phase ^= 1; }
        }
        if (C::ACC == 2) { acc ^= 1; if (acc == 0) acc_phase ^= 1; }
        else acc_phase ^= 1;
      }
    }
  } else {
    // ===== epilogue (both CTAs): warps 2..9; TMEM lane quadrant warp % 4 = 32 of this CTA's 128 pixels, and the two
    // warps of a quadrant (on the same scheduler) take alternate channel chunks: the epilogue is a chain of
    // dependent TMEM load -> convert -> shared store -> TMA store steps, two warps per scheduler hide its latencies.
    // Per 32-channel chunk: tcgen05.ld -> +bias +temb/residual -> bf16 -> this warp's staging buffer (64-byte
    // swizzle, conflict-free) -> one TMA store of the [32 pixels][32 channels] box.  The store clips rows that fall
    // outside the tensor (ragged tiles) and keeps the global writes as full 64-byte segments.
    constexpr int CW = C::CW;
    const int q = warp & 3, grp = (warp - 2) >> 2;
    const int row = q * 32 + lane;
    const int n_l = row / (p.bh * p.bw), rem = row - n_l * (p.bh * p.bw);
    const int y_l = rem / p.bw, x = rem - y_l * p.bw;
    // box origin of this warp inside the tile (lane 0's pixel)
    const int row0 = q * 32, n_w = row0 / (p.bh * p.bw), rem0 = row0 - n_w * (p.bh * p.bw);
    const int y_w = rem0 / p.bw, x_w = rem0 - y_w * p.bw;
    uint8_t* stg_q = smem + C::STAGES * C::STAGE_BYTES + q * (2 * C::NBUF * C::BOX_BYTES + 2048);
    float* colv = reinterpret_cast<float*>(stg_q + 2 * C::NBUF * C::BOX_BYTES);    // [BN] bias (+ temb projection of this image)
    uint8_t* stg = stg_q + grp * C::NBUF * C::BOX_BYTES;                 // this warp's staging boxes
    const uint32_t stg_lane = smem_u32(stg) + lane * (CW * 2);
    const int sw = CW == 64 ? (lane & 7) : ((lane >> 1) & 3);            // 128-byte / 64-byte swizzle of 16-byte pieces
    int acc = 0; uint32_t acc_phase = 0;
    int buf = 0;
    for (int tile = pair; tile < total_tiles; tile += npairs) {
      const int ph = tile / tiles_ph, tl = tile - ph * tiles_ph;
      const int mp = tl / p.n_tiles, nt = tl - mp * p.n_tiles;
      const int mt = 2 * mp + (int)rank;
      const int n_t = (mt / p.tiles_h) * p.bn, y_t = (mt % p.tiles_h) * p.bh;
      const int n = n_t + n_l, y = y_t + y_l;
      const bool valid = mt < p.tiles_m && n < p.GN && y < p.GH;
      const size_t off = (((size_t)n * p.OH + (size_t)y * p.osy + p.ph_ooy[ph]) * p.OW + (size_t)x * p.osx + p.ph_oox[ph]) *
                             p.cout_total + (size_t)nt * C::BN;
      const bf16* addend = p.residual ? p.residual : (p.accumulate ? p.out : nullptr);
      const unsigned vmask = __ballot_sync(0xffffffffu, valid);
      {   // column vector of this quadrant's image, staged while the main loop runs (by the first warp of the pair;
          // named barrier 1 + q joins the quadrant's two warps before and after)
        const int nw = min(n_t + n_w, p.GN - 1);
        asm volatile("bar.sync %0, 64;" ::"r"(1 + q) : "memory");
        if (grp == 0)
          for (int c = lane; c < C::BN; c += 32) {
            float t = p.bias ? to_f(p.bias[nt * C::BN + c]) : 0.f;
            if (p.pn) t += p.pn[(size_t)nw * p.cout_total + nt * C::BN + c];
            colv[c] = t;
          }
        asm volatile("bar.sync %0, 64;" ::"r"(1 + q) : "memory");
      }
      mbar_wait(&tfull_bar[acc], acc_phase);
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + acc * C::BN;
      // one 32-channel chunk of this warp's 32 pixels, accumulator values in r: + bias / temb / residual -> bf16 -> staging
      // box -> TMA store; channel statistics of the stored values
      auto finish_chunk = [&](const int ch, uint32_t (&r)[32]) {
        const int co = nt * C::BN + ch * CW;
        {
          if (lane == 0) bulk_wait_read<C::NBUF - 1>();   // the store that last used this box has read it
          __syncwarp();
          const uint32_t dst = stg_lane + buf * C::BOX_BYTES;
#pragma unroll
          for (int i = 0; i < CW / 8; ++i) {
            const float4 c0 = *reinterpret_cast<const float4*>(colv + ch * CW + i * 8);
            const float4 c1 = *reinterpret_cast<const float4*>(colv + ch * CW + i * 8 + 4);
            float v[8] = {__uint_as_float(r[i * 8]) + c0.x,     __uint_as_float(r[i * 8 + 1]) + c0.y,
                          __uint_as_float(r[i * 8 + 2]) + c0.z, __uint_as_float(r[i * 8 + 3]) + c0.w,
                          __uint_as_float(r[i * 8 + 4]) + c1.x, __uint_as_float(r[i * 8 + 5]) + c1.y,
                          __uint_as_float(r[i * 8 + 6]) + c1.z, __uint_as_float(r[i * 8 + 7]) + c1.w};
            if (addend && valid) {
              float a8[8];
              ldv(addend + off + ch * CW + i * 8, a8);
#pragma unroll
              for (int j = 0; j < 8; ++j) v[j] += a8[j];
            }
            st_shared_v4(dst + ((i ^ sw) << 4), pack_bf16(v[0], v[1]), pack_bf16(v[2], v[3]), pack_bf16(v[4], v[5]),
                         pack_bf16(v[6], v[7]));
          }
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) {
            tma_store_4d(&mapO.m[MP ? ph : 0], stg + buf * C::BOX_BYTES, co, x_w, y_t + y_w, n_t + n_w);
            bulk_commit();
          }
          static_assert(CW == 32, "the statistics pass reads 16 words per staged row");
          if (p.cst && vmask) {
            // channel stats of the STORED (bf16) values for the GroupNorm that reads this tensor: a lane sums two
            // columns of the staged box (one 32-bit word per row) over 16 of the warp's 32 pixel rows - lanes 0-15 the
            // even rows, 16-31 the odd rows: a row is one 64-byte line, so the two halves hit disjoint banks - in packed
            // fp32 pairs; the halves are combined by one shuffle each
            f2_t s2 = pk2(0.f, 0.f), q2 = s2;
            const int half = lane >> 4, l16 = lane & 15;
            const uint32_t base = smem_u32(stg) + buf * C::BOX_BYTES + (l16 & 3) * 4;
            const bool full = vmask == 0xffffffffu;
#pragma unroll
            for (int r0 = 0; r0 < 16; r0 += 8) {       // 8 independent loads in flight, no branches
              uint32_t wv[8];
#pragma unroll
              for (int j = 0; j < 8; ++j) {
                const int r = 2 * (r0 + j) + half;
                const uint32_t swr = CW == 64 ? (r & 7) : ((r >> 1) & 3);
                asm volatile("ld.shared.b32 %0, [%1];" : "=r"(wv[j]) : "r"(base + r * (CW * 2) + (((l16 >> 2) ^ swr) << 4)));
              }
#pragma unroll
              for (int j = 0; j < 8; ++j) {
                f2_t v = bf2(wv[j]);
                if (!full) {                            // rows outside the tensor do not count (warp-uniform branch)
                  const float m = ((vmask >> (2 * (r0 + j) + half)) & 1) ? 1.f : 0.f;
                  v = mul2(v, pk2(m, m));
                }
                s2 = add2(s2, v); q2 = fma2(v, v, q2);
              }
            }
            float s0, s1, q0, q1;
            upk2(s2, s0, s1); upk2(q2, q0, q1);
            s0 += __shfl_xor_sync(0xffffffffu, s0, 16); s1 += __shfl_xor_sync(0xffffffffu, s1, 16);
            q0 += __shfl_xor_sync(0xffffffffu, q0, 16); q1 += __shfl_xor_sync(0xffffffffu, q1, 16);
            float* dst = p.cst + (size_t)(n_t + n_w) * 2 * p.cout_total + co + 2 * l16;
            if (half == 0) {
              atomicAdd(dst, s0); atomicAdd(dst + 1, s1);
              atomicAdd(dst + p.cout_total, q0); atomicAdd(dst + p.cout_total + 1, q1);
            }
          }
          buf ^= 1;
        }
      };
      constexpr int NCH = C::BN / CW;
      if constexpr (SK == 1) {
        // software pipeline: the TMEM load of this warp's next chunk is issued before the current chunk is converted
        // and stored (tcgen05.wait::ld waits for every outstanding load, so the next one is issued right after it)
        constexpr int NIT = (NCH + 1) / 2;
        uint32_t rr[2][32];
        tmem_ld32(taddr + grp * CW, rr[0]);
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
          const int ch = grp + 2 * it;
          if (ch >= NCH) break;
          uint32_t (&r)[32] = rr[it & 1];
          tmem_ld_wait();
          if (ch + 2 < NCH) {
            tmem_ld32(taddr + (ch + 2) * CW, rr[(it + 1) & 1]);
          } else {                                    // that was this warp's last TMEM read of the tile
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster_relaxed(mapa_u32(smem_u32(&tempty_bar[acc]), lead));
          }
          finish_chunk(ch, r);
        }
      } else {
        // split-K: this warp's chunks are [ch_lo, ch_hi); chunk ch belongs to pair ch % SK of the cluster
        constexpr int PER = (NCH + 1) / 2;
        const int ch_lo = grp * PER, ch_hi = ch_lo + PER < NCH ? ch_lo + PER : NCH;
        const uint32_t ring = smem_u32(smem);
        const uint32_t rsw = (uint32_t)(row & 7);
        cluster_arrive(); cluster_wait();             // every CTA of the cluster has seen its accumulator complete: all rings idle
        for (int ch = ch_lo; ch < ch_hi; ++ch) {
          const int owner = ch % SK;
          if (owner == ks) continue;
          uint32_t r[32];
          tmem_ld32(taddr + ch * CW, r);
          tmem_ld_wait();
          // slot (owned-chunk ordinal, sender ordinal) of the owner's ring: [128 rows][32 fp32], 16-byte pieces swizzled by row
          const int slot = (ch / SK) * (SK - 1) + (ks < owner ? ks : ks - 1);
          const uint32_t dst = mapa_u32(ring + (uint32_t)((slot * 128 + row) * 128), (uint32_t)(owner * 2) + rank);
#pragma unroll
          for (int i = 0; i < 8; ++i)
            asm volatile("st.shared::cluster.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(dst + ((i ^ rsw) << 4)), "r"(r[4 * i]),
                         "r"(r[4 * i + 1]), "r"(r[4 * i + 2]), "r"(r[4 * i + 3]) : "memory");
        }
        cluster_arrive(); cluster_wait();             // all partials delivered
        for (int ch = ch_lo; ch < ch_hi; ++ch) {
          if (ch % SK != ks) continue;
          uint32_t r[32];
          tmem_ld32(taddr + ch * CW, r);
          tmem_ld_wait();
#pragma unroll
          for (int s_ = 0; s_ < SK - 1; ++s_) {
            const uint32_t src = ring + (uint32_t)((((ch / SK) * (SK - 1) + s_) * 128 + row) * 128);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              uint32_t v0, v1, v2, v3;
              asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v0), "=r"(v1), "=r"(v2), "=r"(v3) : "r"(src + ((i ^ rsw) << 4)));
              r[4 * i] = __float_as_uint(__uint_as_float(r[4 * i]) + __uint_as_float(v0));
              r[4 * i + 1] = __float_as_uint(__uint_as_float(r[4 * i + 1]) + __uint_as_float(v1));
              r[4 * i + 2] = __float_as_uint(__uint_as_float(r[4 * i + 2]) + __uint_as_float(v2));
              r[4 * i + 3] = __float_as_uint(__uint_as_float(r[4 * i + 3]) + __uint_as_float(v3));
            }
          }
          finish_chunk(ch, r);
        }
      }
      if (C::ACC == 2) { acc ^= 1; if (acc == 0) acc_phase ^= 1; }
      else acc_phase ^= 1;
    }
    if (lane == 0) bulk_wait_read<0>();       // the staging boxes have been read; the global writes complete before the grid does
  }
  if (SK > 1 && warp < 2) {      // the split-K exchange's two cluster barriers count every thread of the cluster
    __syncwarp();
    cluster_arrive(); cluster_wait();
    cluster_arrive(); cluster_wait();
  }
  tc_fence_before();
  cluster_sync_all();          // nobody leaves (or frees TMEM) while the peer may still read its shared memory / TMEM
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc2(tmem_base, C::TMEM_COLS);
  }
}

template <int UN, int NJ, bool MP, int SK>
bool launch2(const CUtensorMap& a0, const CUtensorMap& a1, const CUtensorMap& b, const OutMaps<MP>& o, const Tc2Params& p,
             cudaStream_t st) {
  static bool attr_set = false;
  if (!attr_set) {
    if (cudaFuncSetAttribute(conv_tc2_k<UN, NJ, MP, SK>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg2<UN, NJ>::SMEM) !=
        cudaSuccess) {
      tmap::set_error("cudaFuncSetAttribute(max dynamic smem) failed for conv_tc2_k");
      return false;
    }
    attr_set = true;
  }
  const int tiles = p.nph * p.pair_tiles_m * p.n_tiles;
  const int max_pairs = sm_count() / 2;
  // split-K: one tile per cluster of SK pairs (the exchange's cluster barriers are counted once per CTA)
  const int pairs = SK > 1 ? tiles : (tiles < max_pairs ? tiles : max_pairs);
  launch_pdl(conv_tc2_k<UN, NJ, MP, SK>, dim3(2 * SK * pairs), dim3(320), Cfg2<UN, NJ>::SMEM, st, a0, a1, b, o, p);
  return true;
}

// Split-K factor for a one-phase conv (conv_tc2.cu header): the largest of 4, 2 whose clusters all run in one wave and
// that leaves every pair at least 8 K blocks; 1 = no split.  Only the 320-channel tile (UN = 160, NJ = 2) is instantiated.
int split_k(int tiles, int num_kb, int un, int nj) {
  if (un != 160 || nj != 2 || toggles().no_split_k) return 1;
  const int max_pairs = sm_count() / 2;
  for (int sk = 4; sk >= 2; sk /= 2)
    if (tiles * sk <= max_pairs - max_pairs % sk && num_kb / sk >= 8) return sk;
  return 1;
}

// (UN, NJ) for a channel count: 320 k -> 2 x 160; 160 k -> 1 x 160; 256 k -> 2 x 128; 128 k -> 1 x 128
void pick_tile(int cout, int& un, int& nj) {
  un = nj = 0;
  if (cout % 320 == 0) { un = 160; nj = 2; }
  else if (cout % 160 == 0) { un = 160; nj = 1; }
  else if (cout % 256 == 0) { un = 128; nj = 2; }
  else if (cout % 128 == 0) { un = 128; nj = 1; }
}

}  // namespace

bool conv_tc2_supported(const ConvArgs& a) {
  if (a.dt != DT_BF16) return false;
  if (a.src.c0 % 64 || a.src.c1 % 64 || a.src.c0 == 0) return false;
  int un, nj;
  pick_tile(a.cout, un, nj);
  if (!un) return false;
  if (a.ksize != 1 && a.ksize != 3) return false;
  int bw, bh, bn;
  if (a.mode == CONV_UP2_DGRAD) {
    if (a.ksize != 3 || a.src.c1 || (a.hin & 1) || (a.win & 1) || a.hout * 2 != a.hin || a.wout * 2 != a.win) return false;
    return tile_geometry(a.hout, a.wout, bw, bh, bn) && bw * bh >= 32;
  }
  if (a.mode == CONV_DGRAD_S2 || a.mode == CONV_UP2) {
    if (a.ksize != 3 || a.src.c1) return false;
    if (a.hout != 2 * a.hin || a.wout != 2 * a.win) return false;
    return tile_geometry(a.hin, a.win, bw, bh, bn) && bw * bh >= 32;
  }
  if (a.stride == 2) {
    if (a.ksize != 3 || a.src.c1 || (a.hin & 1) || (a.win & 1) || a.hout * 2 != a.hin || a.wout * 2 != a.win) return false;
  } else if (a.stride != 1 || a.hout != a.hin || a.wout != a.win) {
    return false;
  }
  return tile_geometry(a.hout, a.wout, bw, bh, bn) && bw * bh >= 32;      // a warp's 32 pixels lie inside one image
}

int conv_tc2(const ConvArgs& a, cudaStream_t st) {
  Tc2Params p;
  memset(&p, 0, sizeof p);
  int un, nj;
  pick_tile(a.cout, un, nj);
  const bool s2d = a.mode == CONV_DGRAD_S2, up2 = a.mode == CONV_UP2, up2d = a.mode == CONV_UP2_DGRAD;
  const bool s2f = up2d || (a.mode == CONV_FPROP && a.stride == 2);      // source read through the 5-D parity view
  const int gh = (s2d || up2) ? a.hin : a.hout, gw = (s2d || up2) ? a.win : a.wout;
  tile_geometry(gh, gw, p.bw, p.bh, p.bn);
  p.c0 = a.src.c0; p.ctot = a.src.c(); p.c0_blocks = a.src.c0 / 64; p.c_blocks = p.ctot / 64;
  p.s2 = s2f;
  p.tiles_h = (gh + p.bh - 1) / p.bh;
  p.tiles_m = p.tiles_h * ((a.n + p.bn - 1) / p.bn);
  p.pair_tiles_m = (p.tiles_m + 1) / 2;
  p.n_tiles = a.cout / (un * nj);
  p.GH = gh; p.GN = a.n;
  p.bias = (const bf16*)a.bias; p.pn = a.pn; p.residual = (const bf16*)a.residual; p.out = (bf16*)a.out;
  p.accumulate = a.accumulate;
  p.cst = a.cst;
  CUtensorMap m0, m1, mb;
  bool ok = true;
  if (s2f) ok = act_map_s2(a.src.p0, a.n, a.hin, a.win, a.src.c0, p.bw, p.bh, p.bn, &m0);
  else ok = act_map(a.src.p0, a.n, a.hin, a.win, a.src.c0, p.bw, p.bh, p.bn, &m0);
  m1 = m0;
  if (ok && a.src.c1) ok = act_map(a.src.p1, a.n, a.hin, a.win, a.src.c1, p.bw, p.bh, p.bn, &m1);
  const uint64_t wk = (uint64_t)(up2 ? 4 : up2d ? 16 : a.ksize * a.ksize) * p.ctot;     // K of the weight matrix
  if (ok) ok = mat_map(a.w, (uint64_t)(up2 ? 4 : 1) * a.cout, wk, un / 2, &mb);
  if (!ok) return -1;
  // phases: taps, weight rows and output parity of each sub-pixel conv of this launch (one phase for a plain conv)
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
    // output pixel (2y+py, 2x+px) <- low-resolution pixels (y+dy, x+dx), dy = a-1+py, dx = b-1+px, through the pre-summed
    // weights Wp[phase] (kernels.h): rows [phase cout, (phase + 1) cout) of one [4 cout][4 c] matrix
    p.osy = p.osx = 2;
    for (int ph = 0; ph < 4; ++ph) {
      const int py = ph >> 1, px = ph & 1;
      for (int t = 0; t < 4; ++t) add_tap((t >> 1) - 1 + py, (t & 1) - 1 + px, 0, 0, t);
      end_phase(ph * a.cout, py, px);
    }
  } else if (up2d) {
    // g_in(y, x) = sum over (phase, tap) of WpT[..][q] g(2 (y - dy) + py, 2 (x - dx) + px): 16 taps on the parity view
    for (int q = 0; q < 16; ++q) {
      const int py = q >> 3, px = (q >> 2) & 1, ta = (q >> 1) & 1, tb = q & 1;
      add_tap(1 - ta - py, 1 - tb - px, py, px, q);
    }
    end_phase(0, 0, 0);
  } else if (s2d) {
    // output pixel (2y'+py, 2x'+px) <- taps r' with (py + r' - 1) even: py=0: r'=1 (dy 0); py=1: r'=0 (dy 0), r'=2 (dy +1).
    // Phases in order of decreasing tap count (4, 2, 2, 1): the round-robin tile walk then mixes long and short tiles
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
        else add_tap(r == 0 ? -1 : 0, s_ == 0 ? -1 : 0, r == 1 ? 0 : 1, s_ == 1 ? 0 : 1, r * a.ksize + s_);   // input row 2y + r - 1 = 2(y + dy) + py
      }
    end_phase(0, 0, 0);
  }
  // output view of each phase: (c, x, y, n) with pixel strides osx/osy from pixel (ooy, oox); box = one warp's
  // [32 pixels][32 channels], 64-byte swizzle
  OutMaps<true> mo;
  for (int ph = 0; ph < p.nph; ++ph) {
    const int bwb = p.bw < 32 ? p.bw : 32, bhb = 32 / bwb;
    const size_t C2 = (size_t)a.cout * 2;
    uint64_t dims[4] = {(uint64_t)a.cout, (uint64_t)gw, (uint64_t)gh, (uint64_t)a.n};
    uint64_t str[3] = {(uint64_t)p.osx * C2, (uint64_t)p.osy * a.wout * C2, (uint64_t)a.hout * a.wout * C2};
    const uint32_t cw = 32;        // Cfg2::CW
    uint32_t box[4] = {cw, (uint32_t)bwb, (uint32_t)bhb, 1};
    const char* base = (const char*)a.out + ((size_t)p.ph_ooy[ph] * a.wout + p.ph_oox[ph]) * C2;
    if (!get_map(base, 4, dims, str, box, &mo.m[ph], 2 * (int)cw)) return -1;
  }
  bool r;
  if (p.nph == 1) {
    OutMaps<false> m1p;
    m1p.m[0] = mo.m[0];
    const int sk = (a.mode == CONV_FPROP && a.stride == 1) ? split_k(p.pair_tiles_m * p.n_tiles, ntaps * p.c_blocks, un, nj) : 1;
    if (sk == 4) r = launch2<160, 2, false, 4>(m0, m1, mb, m1p, p, st);
    else if (sk == 2) r = launch2<160, 2, false, 2>(m0, m1, mb, m1p, p, st);
    else
      r = un == 160 ? (nj == 2 ? launch2<160, 2, false, 1>(m0, m1, mb, m1p, p, st) : launch2<160, 1, false, 1>(m0, m1, mb, m1p, p, st))
                    : (nj == 2 ? launch2<128, 2, false, 1>(m0, m1, mb, m1p, p, st) : launch2<128, 1, false, 1>(m0, m1, mb, m1p, p, st));
  } else {
    for (int ph = p.nph; ph < 4; ++ph) mo.m[ph] = mo.m[0];
    r = un == 160 ? (nj == 2 ? launch2<160, 2, true, 1>(m0, m1, mb, mo, p, st) : launch2<160, 1, true, 1>(m0, m1, mb, mo, p, st))
                  : (nj == 2 ? launch2<128, 2, true, 1>(m0, m1, mb, mo, p, st) : launch2<128, 1, true, 1>(m0, m1, mb, mo, p, st));
  }
  return r ? 1 : -1;
}

// Few output tiles (deep UNet levels: 1280 channels on 8 x 8 or 16 x 16 pixels give 8 / 32 pair tiles for 74 CTA
// pairs): every tile runs in one wave either way, so the step time is ONE tile's time, and the single-CTA 128 x 160
// tile has a quarter of the pair tile's MMAs (at 57 % of the pair's MMA rate: 0.44 of its time).  The single-CTA
// kernel is preferred while all of its tiles still fit one wave.  PULSE_CONV_1CTA_TILES overrides the bound
// (single-CTA tiles; 0 = never).
static int one_cta_tile_bound() { return toggles().conv_1cta_tiles >= 0 ? toggles().conv_1cta_tiles : sm_count(); }
// split-K factor conv_tc2 would use for this conv (1: none)
static int split_k_of(const ConvArgs& a) {
  if (a.mode != CONV_FPROP || a.stride != 1 || !conv_tc2_supported(a)) return 1;
  int un, nj, bw, bh, bn;
  pick_tile(a.cout, un, nj);
  if (!tile_geometry(a.hout, a.wout, bw, bh, bn)) return 1;
  const int tiles_m = ((a.hout + bh - 1) / bh) * ((a.n + bn - 1) / bn);
  return split_k(((tiles_m + 1) / 2) * (a.cout / (un * nj)), a.ksize * a.ksize * (a.src.c() / 64), un, nj);
}
static bool prefer_1cta(const ConvArgs& a) {
  if (!conv_tc_supported(a)) return false;
  if (split_k_of(a) > 1) return false;       // few tiles and a long K: the pair kernel splits K over a cluster instead
  const bool s2d = a.mode == CONV_DGRAD_S2 || a.mode == CONV_UP2;      // pixel grid = the low-resolution side
  int bw, bh, bn;
  if (!tile_geometry(s2d ? a.hin : a.hout, s2d ? a.win : a.wout, bw, bh, bn)) return false;
  const int gh = s2d ? a.hin : a.hout;
  const long long tiles_m = (long long)((gh + bh - 1) / bh) * ((a.n + bn - 1) / bn) * (s2d ? 4 : 1);      // 4 phases per launch
  const long long tiles = tiles_m * (a.cout / (a.cout % 160 == 0 ? 160 : 128));      // its N tiles are 160 (or 128) wide
  return tiles <= one_cta_tile_bound();
}
// a.kernel: CONV_K_AUTO picks by tile count (above); CONV_K_PAIR / CONV_K_1CTA force one kernel where it applies
static bool use_pair(const ConvArgs& a) {
  if (!conv_tc2_supported(a)) return false;
  if (a.kernel == CONV_K_PAIR || !conv_tc_supported(a)) return true;
  if (a.kernel == CONV_K_1CTA || toggles().conv_1cta) return false;
  return !prefer_1cta(a);
}
bool conv_emits_stats(const ConvArgs& a) { return use_pair(a) && (a.mode == CONV_FPROP || a.mode == CONV_UP2) && !a.accumulate; }
bool conv_tc_any_supported(const ConvArgs& a) {
  if (a.kernel == CONV_K_PAIR) return conv_tc2_supported(a);
  if (a.kernel == CONV_K_1CTA) return conv_tc_supported(a);
  return conv_tc2_supported(a) || conv_tc_supported(a);
}
int conv_tc_any(const ConvArgs& a, cudaStream_t st) {
  if (use_pair(a)) return conv_tc2(a, st);
  return conv_tc(a, st);
}

}  // namespace pulse

// norm_fused.cu - GroupNorm + SiLU backward in ONE pass over memory (SURVEY.md 8c item 1, bf16 tensors).
//   g_y = g_a SiLU'(y); S1[c] = sum_pix g_y; S2[c] = sum_pix g_y xhat; A = mean_S gamma g_y; B = mean_S gamma g_y xhat;
//   g_x = r (gamma g_y - A - xhat B) [+ add];  dgamma += S2, dbeta += S1
// The two-kernel form (norm.cu: gn_bwd_stats_k, then gn_bwd_apply_k) reads x and g_a twice and pays two launches
// with their ramps; at 10 MB per tensor those ramps are most of the time.  GroupNorm groups are independent, so a
// work item here is (image, slice of whole groups): Cs = lcm(channels per group, 8) channels, i.e. 16-byte
// aligned channel vectors.  A CLUSTER of CL CTAs owns one item; each CTA keeps its 1/CL of the pixels of x and g_a
// resident in shared memory (TMA boxes [BR pixels][Cs channels], no swizzle: a pixel's Cs channels are one row):
//   phase 1  as the boxes land: the per-channel S1, S2; CTA reduction through shared memory, cluster reduction
//            through distributed shared memory
//   phase 2  g_x from the resident x and g_a: no second read (g_y is recomputed in fp32: keeping it in shared
//            memory as bf16 would add a rounding the two-kernel form does not have); `add` (the shortcut
//            gradient) streams in through a per-thread cp.async ring started before the reductions.
//            (Measured and rejected in round 2: keeping g_y as fp32 IN PLACE of the x / g_a it came from and reading x
//            again from L2 in phase 2, three pixels ahead in registers - it halves the special-function work, but a
//            thread has only ~10 pixels per phase, too few to hide the L2 latency: 16.4 vs 15.9 us per launch.)
// Falls back (returns 0) when a slice of one image does not fit into 8 CTAs' shared memory or the channel split
// does not fall on slice boundaries; norm.cu then runs the two-kernel form.
#include <cuda.h>

#include <cstdlib>

#include "common.cuh"
#include "kernels.h"
#include "sm100.cuh"
#include "tmap.h"

namespace pulse {

namespace {

using namespace sm100;

constexpr int MAXBOX = 16;     // TMA boxes per tensor per CTA
constexpr int ED = 2;          // depth of the per-thread cp.async ring for `add`
constexpr int NP = 8;          // partial sums per value in the second stage of the CTA reduction
constexpr int MAXCS = 120;     // widest slice (channels per group 30 -> lcm(30, 8))

struct GnfParams {
  int c0, c1, hw, G, Cs, CL, ppc, BR, nbox, nrow, br_shift;   // BR = 1 << br_shift
  const bf16* gamma; const bf16* beta; const float* mr;
  float* dgamma; float* dbeta;
  const bf16* add; bf16* dst0; bf16* dst1; int dc0, acc0, acc1;
  float* cs0; float* cs1;
  int data_bytes, red_floats;
  int act;                       // 1: GroupNorm + SiLU, 0: plain GroupNorm (g_y = g_a)
};

__device__ __forceinline__ void lds8(const uint8_t* p, float (&o)[8]) { ldv(reinterpret_cast<const bf16*>(p), o); }

__device__ __forceinline__ float ex2_(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float rcp_(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
// SiLU'(y) = s + y s (1 - s), s = 1 / (1 + 2^(-y log2 e)), of the pair y = x sc + sh; also returns nothing else: the
// MUFU work (ex2, rcp) is per lane, everything around it is packed
__device__ __forceinline__ f2_t silu_grad2(f2_t y, f2_t nl2e, f2_t one, f2_t mone) {
  const f2_t t = mul2(y, nl2e);
  float t0, t1;
  upk2(t, t0, t1);
  const f2_t d = add2(pk2(ex2_(t0), ex2_(t1)), one);
  float d0, d1;
  upk2(d, d0, d1);
  const f2_t sg = pk2(rcp_(d0), rcp_(d1));
  return fma2(mul2(y, sg), fma2(sg, mone, one), sg);
}

// sum v[K] over the `nrow` threads that share a channel vector; result[j], j < K * tpp (layout [k][Cs]) is returned
// to every thread through `out` (shared memory, K * Cs floats).  Whole CTA; `red` holds nrow * K * Cs + NP * K * Cs floats.
template <int K>
__device__ __forceinline__ void cta_reduce(const float (&v)[K][8], bool active, int row, int vec, int nrow, int Cs,
                                           float* red, float* out) {
  const int W = K * Cs, tid = threadIdx.x;
  if (active) {
#pragma unroll
    for (int k = 0; k < K; ++k) {
      float4* d = reinterpret_cast<float4*>(red + (size_t)row * W + k * Cs + vec * 8);
      d[0] = make_float4(v[k][0], v[k][1], v[k][2], v[k][3]);
      d[1] = make_float4(v[k][4], v[k][5], v[k][6], v[k][7]);
    }
  }
  __syncthreads();
  float* red2 = red + (size_t)nrow * W;
  for (int u = tid; u < NP * W; u += blockDim.x) {
    const int part = u / W, j = u - part * W;
    float t = 0.f;
    for (int r = part; r < nrow; r += NP) t += red[(size_t)r * W + j];
    red2[u] = t;
  }
  __syncthreads();
  if (tid < W) {
    float t = 0.f;
#pragma unroll
    for (int q = 0; q < NP; ++q) t += red2[q * W + tid];
    out[tid] = t;
  }
  __syncthreads();
}

// ACT: 1 = GroupNorm + SiLU, 0 = plain GroupNorm (g_y = g_a); a template parameter because the phase loops are bound by
// instruction issue (a run-time select in them cost 2 % of the kernel)
template <int ACT>
__global__ void __launch_bounds__(512, 1)
gn_bwd_fused_k(const __grid_constant__ CUtensorMap mapX0, const __grid_constant__ CUtensorMap mapX1,
               const __grid_constant__ CUtensorMap mapG, const GnfParams p) {
  extern __shared__ uint8_t smem_raw[];
  __shared__ uint64_t fullx[MAXBOX], fullg[MAXBOX];
  __shared__ float tot[2 * MAXCS];          // S1 | S2 of the slice: this CTA, then the whole cluster
  __shared__ float grpAB[2][MAXCS / 8];     // A, B per group of the slice
  uint8_t* base = smem_raw + ((128 - (smem_u32(smem_raw) & 127)) & 127);
  uint8_t* xs = base;
  uint8_t* gs = xs + p.data_bytes;
  float* red = reinterpret_cast<float*>(gs + p.data_bytes);
  float* cl = red + p.red_floats;                                  // [CL][2 Cs]: every CTA's S1 | S2
  uint8_t* ering = reinterpret_cast<uint8_t*>(cl + p.CL * 2 * p.Cs);

  const int tid = threadIdx.x, Cs = p.Cs, tpp = Cs >> 3, nrow = p.nrow, nthr = nrow * tpp;
  const uint32_t rank = cluster_ctarank();
  const int slice = blockIdx.x / p.CL, n = blockIdx.y;
  const int C = p.c0 + p.c1, chs = slice * Cs, cpg = C / p.G, rb = Cs * 2;
  const bool active = tid < nthr;
  const int row = active ? tid / tpp : 0, vec = active ? tid - row * tpp : 0, ch = chs + vec * 8;
  const int prow = n * p.hw + (int)rank * p.ppc;       // first pixel (row of the [n hw][C] matrices) of this CTA
  if (tid == 0) {
    prefetch_tmap(&mapX0); prefetch_tmap(&mapX1); prefetch_tmap(&mapG);
    for (int b = 0; b < p.nbox; ++b) { mbar_init(&fullx[b], 1); mbar_init(&fullg[b], 1); }
    fence_barrier_init();
    // x is a tensor of the FORWARD pass: not written by the previous kernel, so its boxes are requested before the
    // dependency wait and stream in while that kernel drains
    const bool lo = chs < p.c0;
    for (int b = 0; b < p.nbox; ++b) {
      mbar_expect_tx(&fullx[b], (uint32_t)(p.BR * rb));
      tma_load_2d(xs + (size_t)b * p.BR * rb, lo ? &mapX0 : &mapX1, &fullx[b], lo ? chs : chs - p.c0, prow + b * p.BR);
    }
  }
  cluster_arrive();                          // #1: waited on before the first remote shared-memory write
  float sc[8], sh[8], rr[8], mr[8];
  {
    float gav[8], bev[8];
    ldv(p.gamma + ch, gav); ldv(p.beta + ch, bev);
    int g = ch / cpg, rem = ch - g * cpg;        // one division; the 8 channels then walk the groups
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const float mu = p.mr[(size_t)n * 2 * p.G + g], r = p.mr[(size_t)n * 2 * p.G + p.G + g];
      rr[i] = r; mr[i] = mu * r;
      sc[i] = r * gav[i]; sh[i] = bev[i] - mr[i] * gav[i];
      if (++rem == cpg) { rem = 0; ++g; }
    }
  }
  pdl_wait();
  pdl_launch_dependents();
  if (tid == 0)
    for (int b = 0; b < p.nbox; ++b) {
      mbar_expect_tx(&fullg[b], (uint32_t)(p.BR * rb));
      tma_load_2d(gs + (size_t)b * p.BR * rb, &mapG, &fullg[b], chs, prow + b * p.BR);
    }
  __syncthreads();                           // barrier initialisation is visible to every thread

  // ---- phase 1 ------------------------------------------------------------------------------------------
  float S[2][8];
  f2_t S2[2][4], sc2[4], sh2[4], rr2[4], nmr2[4];
  const f2_t nl2e = pk2(-1.4426950408889634f, -1.4426950408889634f), one = pk2(1.0f, 1.0f), mone = pk2(-1.0f, -1.0f);
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    S2[0][j] = S2[1][j] = pk2(0.f, 0.f);
    sc2[j] = pk2(sc[2 * j], sc[2 * j + 1]); sh2[j] = pk2(sh[2 * j], sh[2 * j + 1]);
    rr2[j] = pk2(rr[2 * j], rr[2 * j + 1]); nmr2[j] = pk2(-mr[2 * j], -mr[2 * j + 1]);
  }
  if (active) {
    int waited = 0;
    int off = row * rb + vec * 16;
    const int step = nrow * rb;
    for (int pl = row; pl < p.ppc; pl += nrow, off += step) {
      const int b = pl >> p.br_shift;
      while (waited <= b) { mbar_wait(&fullx[waited], 0); mbar_wait(&fullg[waited], 0); ++waited; }
      const uint4 xw = *reinterpret_cast<const uint4*>(xs + off), gw = *reinterpret_cast<const uint4*>(gs + off);
      const uint32_t xv[4] = {xw.x, xw.y, xw.z, xw.w}, gv[4] = {gw.x, gw.y, gw.z, gw.w};
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const f2_t x = bf2(xv[j]);
        const f2_t gy = ACT ? mul2(bf2(gv[j]), silu_grad2(fma2(x, sc2[j], sh2[j]), nl2e, one, mone)) : bf2(gv[j]);
        S2[0][j] = add2(S2[0][j], gy);
        S2[1][j] = fma2(gy, fma2(x, rr2[j], nmr2[j]), S2[1][j]);
      }
    }
  }
#pragma unroll
  for (int j = 0; j < 4; ++j) { upk2(S2[0][j], S[0][2 * j], S[0][2 * j + 1]); upk2(S2[1][j], S[1][2 * j], S[1][2 * j + 1]); }
  // `add` ring: the first ED pixels of this thread are requested now, their latency hides behind the reductions
  const size_t gpix0 = (size_t)prow;
  const uint32_t eslot = smem_u32(ering) + (uint32_t)tid * 16;
  if (p.add) {
#pragma unroll
    for (int d = 0; d < ED; ++d) {
      const int pl = row + d * nrow;
      if (active && pl < p.ppc) cp_async16(eslot + (uint32_t)d * nthr * 16, p.add + (gpix0 + pl) * C + ch);
      cp_async_commit();
    }
  }
  cta_reduce<2>(S, active, row, vec, nrow, Cs, red, tot);
  // cluster reduction: every CTA writes its 2 Cs sums into slot [rank] of every CTA of the cluster
  cluster_wait();                            // #1: every CTA of the cluster is running
  if (tid < 2 * Cs) {
    const float v = tot[tid];
    const uint32_t a = smem_u32(cl + (size_t)rank * 2 * Cs + tid);
    for (int q = 0; q < p.CL; ++q) st_cluster_f32(mapa_u32(a, (uint32_t)q), v);
  }
  cluster_arrive();                          // #2 (release): the remote writes above ...
  cluster_wait();                            //    (acquire): ... are visible to everyone
  if (tid < 2 * Cs) {
    float t = 0.f;
    for (int q = 0; q < p.CL; ++q) t += cl[(size_t)q * 2 * Cs + tid];
    tot[tid] = t;
    if (rank == 0) atomicAdd((tid < Cs ? p.dbeta + chs + tid : p.dgamma + chs + (tid - Cs)), t);
  }
  __syncthreads();
  if (tid < Cs / cpg) {                      // A, B of the groups of this slice
    float a = 0.f, b = 0.f;
    for (int c = tid * cpg; c < (tid + 1) * cpg; ++c) {
      const float ga = to_f(p.gamma[chs + c]);
      a = fmaf(ga, tot[c], a); b = fmaf(ga, tot[Cs + c], b);
    }
    const float inv = 1.0f / ((float)cpg * (float)p.hw);
    grpAB[0][tid] = a * inv; grpAB[1][tid] = b * inv;
  }
  __syncthreads();
  // ---- phase 2 ------------------------------------------------------------------------------------------
  float sum[1][8];
  f2_t nk2[4], nk3[4], sum2[4];        // -A r, -B r per channel pair
  {
    float k2[8], k3[8];
    int g = (vec * 8) / cpg, rem = vec * 8 - g * cpg;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      k2[i] = grpAB[0][g] * rr[i];
      k3[i] = grpAB[1][g] * rr[i];
      if (++rem == cpg) { rem = 0; ++g; }
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      nk2[j] = pk2(-k2[2 * j], -k2[2 * j + 1]); nk3[j] = pk2(-k3[2 * j], -k3[2 * j + 1]);
      sum2[j] = pk2(0.f, 0.f);
    }
  }
  const bool first = ch < p.dc0;
  bf16* dst = first ? p.dst0 : p.dst1;
  const int dC = first ? p.dc0 : C - p.dc0, dch = first ? ch : ch - p.dc0;
  const int acc = first ? p.acc0 : p.acc1;
  if (active) {
    int it = 0;
    int off = row * rb + vec * 16;
    const int step = nrow * rb;
    bf16* d = dst + (gpix0 + row) * dC + dch;
    const size_t dstep = (size_t)nrow * dC;
    const bf16* ap = p.add ? p.add + (gpix0 + row + ED * nrow) * C + ch : nullptr;      // the pixel ED passes ahead
    const size_t astep = (size_t)nrow * C;
    for (int pl = row; pl < p.ppc; pl += nrow, ++it, off += step, d += dstep) {
      const uint4 xw = *reinterpret_cast<const uint4*>(xs + off), gw = *reinterpret_cast<const uint4*>(gs + off);
      const uint32_t xv[4] = {xw.x, xw.y, xw.z, xw.w}, gv[4] = {gw.x, gw.y, gw.z, gw.w};
      f2_t o[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) {          // g_y again, in fp32 (keeping it in shared memory would round it to bf16)
        const f2_t x = bf2(xv[j]);
        const f2_t gy = ACT ? mul2(bf2(gv[j]), silu_grad2(fma2(x, sc2[j], sh2[j]), nl2e, one, mone)) : bf2(gv[j]);
        o[j] = fma2(fma2(x, rr2[j], nmr2[j]), nk3[j], fma2(sc2[j], gy, nk2[j]));
      }
      if (p.add) {
        cp_async_wait<ED - 1>();             // the oldest outstanding request (this pixel's) has landed
        const uint32_t sidx = (uint32_t)(it & (ED - 1)) * nthr * 16;
        const uint4 ew = *reinterpret_cast<const uint4*>(ering + tid * 16 + sidx);
        if (pl + ED * nrow < p.ppc) cp_async16(eslot + sidx, ap);        // refill the slot just read
        cp_async_commit();
        ap += astep;
        o[0] = add2(o[0], bf2(ew.x)); o[1] = add2(o[1], bf2(ew.y));
        o[2] = add2(o[2], bf2(ew.z)); o[3] = add2(o[3], bf2(ew.w));
      }
#pragma unroll
      for (int j = 0; j < 4; ++j) sum2[j] = add2(sum2[j], o[j]);
      if (acc) {
        const uint4 fw = *reinterpret_cast<const uint4*>(d);
        o[0] = add2(o[0], bf2(fw.x)); o[1] = add2(o[1], bf2(fw.y));
        o[2] = add2(o[2], bf2(fw.z)); o[3] = add2(o[3], bf2(fw.w));
      }
      uint4 ov;
      float a, b;
      upk2(o[0], a, b); ov.x = pack_bf16(a, b);
      upk2(o[1], a, b); ov.y = pack_bf16(a, b);
      upk2(o[2], a, b); ov.z = pack_bf16(a, b);
      upk2(o[3], a, b); ov.w = pack_bf16(a, b);
      *reinterpret_cast<uint4*>(d) = ov;
    }
  }
#pragma unroll
  for (int j = 0; j < 4; ++j) upk2(sum2[j], sum[0][2 * j], sum[0][2 * j + 1]);
  if (p.cs0 || p.cs1) {        // per-(image, channel) sums of what this launch adds to dst0 / dst1
    cta_reduce<1>(sum, active, row, vec, nrow, Cs, red, tot);
    if (tid < Cs) {
      const int c = chs + tid;
      if (c < p.dc0) { if (p.cs0) atomicAdd(p.cs0 + (size_t)n * p.dc0 + c, tot[tid]); }
      else if (p.cs1) atomicAdd(p.cs1 + (size_t)n * (C - p.dc0) + (c - p.dc0), tot[tid]);
    }
  }
}

}  // namespace

static int gcd_(int a, int b) { while (b) { const int t = a % b; a = b; b = t; } return a; }

// One launch, or 0 when the shape is not covered (the caller then runs the two-kernel form).
int gn_bwd_fused(const void* g_a, Cat x, int n, int hw, int groups, const void* gamma, const void* beta, const float* mr,
                 const void* add, void* dst0, int dc0, int acc0, void* dst1, int acc1, float* dgamma, float* dbeta,
                 float* cs0, float* cs1, cudaStream_t st, bool fwd_data_ready, int act) {
  static bool enabled = !toggles().no_gn_fused;
  if (!enabled) return 0;
  const int C = x.c();
  if (groups <= 0 || C % groups) return 0;
  const int cpg = C / groups;
  const int Cs = cpg / gcd_(cpg, 8) * 8;               // lcm(cpg, 8)
  if (Cs > MAXCS || C % Cs || x.c0 % Cs || dc0 % Cs || (x.c1 && x.c1 % 8) || x.c0 % 8) return 0;
  if ((long long)n * hw >= (1LL << 31) / Cs) return 0;
  const int tpp = Cs / 8, rb = Cs * 2;
  const int slices = C / Cs;
  const int budget = 227 * 1024 - 128 - 2048;          // dynamic shared memory: alignment slack, static arrays
  GnfParams p;
  int CL = 0, smem = 0;
  for (int cl = 1; cl <= 8; cl *= 2) {
    if (hw % cl) break;
    const int ppc = hw / cl;
    int nrow = 512 / tpp;
    if (nrow > ppc) nrow = ppc;
    int BR = ppc;
    while (BR > 128 && BR % 2 == 0) BR /= 2;
    while (ppc / BR > MAXBOX && BR * 2 <= 256 && ppc % (BR * 2) == 0) BR *= 2;
    if (BR > 256 || ppc % BR || ppc / BR > MAXBOX || (BR * rb) % 128 || (BR & (BR - 1))) continue;
    const int data = ppc * rb;
    const int red = nrow * 2 * Cs + NP * 2 * Cs;
    const int need = 2 * data + (red + cl * 2 * Cs) * 4 + (add ? ED * nrow * tpp * 16 : 0);
    if (need > budget) continue;
    // the smallest cluster that fits; a larger one only while the grid would leave most SMs idle
    const long long ctas = (long long)n * slices * cl;
    CL = cl; smem = need + 128;
    p.br_shift = 0;
    while ((1 << p.br_shift) < BR) ++p.br_shift;
    p.ppc = ppc; p.BR = BR; p.nbox = ppc / BR; p.nrow = nrow; p.data_bytes = data; p.red_floats = red;
    if (ctas * 4 >= 3LL * tmap::sm_count() || ppc / 2 < 4 * nrow) break;
  }
  if (!CL) return 0;
  p.c0 = x.c0; p.c1 = x.c1; p.hw = hw; p.G = groups; p.Cs = Cs; p.CL = CL;
  p.gamma = (const bf16*)gamma; p.beta = (const bf16*)beta; p.mr = mr; p.dgamma = dgamma; p.dbeta = dbeta;
  p.add = (const bf16*)add; p.dst0 = (bf16*)dst0; p.dst1 = (bf16*)dst1; p.dc0 = dc0; p.acc0 = acc0; p.acc1 = acc1;
  p.cs0 = cs0; p.cs1 = cs1; p.act = act;
  CUtensorMap mx0, mx1, mg;
  const uint64_t rows = (uint64_t)n * hw;
  auto mk = [&](const void* ptr, int c, CUtensorMap* m) {
    const uint64_t dims[2] = {(uint64_t)c, rows}, str[1] = {(uint64_t)c * 2};
    const uint32_t box[2] = {(uint32_t)Cs, (uint32_t)p.BR};
    return tmap::get_map(ptr, 2, dims, str, box, m, 0);
  };
  if (!mk(x.p0, x.c0, &mx0)) return 0;
  if (x.c1) { if (!mk(x.p1, x.c1, &mx1)) return 0; } else mx1 = mx0;
  if (!mk(g_a, C, &mg)) return 0;
  static bool attr = false;
  if (!attr) {
    if (cudaFuncSetAttribute(gn_bwd_fused_k<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 2048) != cudaSuccess ||
        cudaFuncSetAttribute(gn_bwd_fused_k<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 2048) != cudaSuccess) {
      cudaGetLastError();
      enabled = false;
      return 0;
    }
    attr = true;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(slices * CL, n); cfg.blockDim = dim3((p.nrow * tpp + 31) & ~31);
  cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = CL; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[1].val.programmaticStreamSerializationAllowed = (pdl_enabled() && fwd_data_ready) ? 1 : 0;
  cfg.attrs = at; cfg.numAttrs = 2;
  const cudaError_t e = act ? cudaLaunchKernelEx(&cfg, gn_bwd_fused_k<1>, mx0, mx1, mg, p)
                            : cudaLaunchKernelEx(&cfg, gn_bwd_fused_k<0>, mx0, mx1, mg, p);
  if (e != cudaSuccess) { cudaGetLastError(); return 0; }
  return 1;
}

}  // namespace pulse

// norm.cu - fused GroupNorm + SiLU forward / backward on NHWC tensors, single or dual
// source (virtual concat).  SURVEY.md 8c item 1:
//   fwd: mu, var per (n,group) (biased), r = rsqrt(var+eps), xhat = (x-mu) r,
//        y = gamma xhat + beta, a = y sigmoid(y)
//   bwd: g_y = g_a SiLU'(y); dgamma = sum g_y xhat; dbeta = sum g_y; q = g_y gamma;
//        A = mean_S q; B = mean_S q xhat; g_x = r (q - A - xhat B)
// HBM-bound, so the design is about passes over memory:
//  * Statistics travel as PER-(image, channel) sums [n][2][C] fp32 ("channel stats").  Group
//    sums are formed from them in a few hundred cycles of kernel prologue, which makes groups
//    that are not 16-byte aligned (10/20/30/60 channels) or that straddle the h|skip boundary
//    (960 = 640|320) irrelevant, and lets the PRODUCER of a tensor (a conv epilogue, or
//    chan_stats_k for tensors that enter from outside) supply them: the forward is then a
//    single read + write pass, and a tensor consumed by two GroupNorm sites (an encoder output
//    that is also a cached skip) has its statistics computed once.
//  * The backward needs per-(image, channel) sums of g_y and g_y xhat: one reduction pass
//    (gn_bwd_stats_k), then one apply pass that also emits the per-(image, channel) sums of the
//    gradient it writes (bias / temb-projection gradients need exactly those: no separate
//    column-sum pass over the tensor).
//  * Thread layout: a thread owns one 16-byte channel vector and walks pixels, so a CTA reads
//    whole contiguous pixel rows (fully coalesced), per-channel partials live in registers,
//    cross-CTA reduction is one fp32 atomic per channel per CTA (<= ~74-way per address).
//  * Memory-level parallelism without registers: the apply / backward kernels stream their inputs through a
//    shared-memory ring filled by bulk asynchronous copies (cp.async.bulk + mbarrier, one elected thread issues).
//    The first stages are requested at kernel entry, BEFORE the statistics prologue, so DRAM latency overlaps
//    the prologue, and a 10 MB tensor spread over 148 CTAs is entirely in flight at once.
#include <type_traits>

#include "common.cuh"
#include "kernels.h"
#include "sm100.cuh"

namespace pulse {

static int g_num_sms = 0;
static int num_sms() {
  if (!g_num_sms) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&g_num_sms, cudaDevAttrMultiProcessorCount, dev);
    if (g_num_sms <= 0) g_num_sms = 148;
  }
  return g_num_sms;
}

RowPlan row_plan(int dt, int hw, int c, int n, int max_threads) {
  RowPlan p;
  const int vec = dt == DT_F32 ? 4 : 8;
  p.tpr = c / vec;
  p.rows = p.tpr >= max_threads ? 1 : max_threads / p.tpr;
  if (p.rows > hw) p.rows = hw;
  // ~2 CTAs per SM over the whole grid, at least 4 pixels per thread row (one unrolled batch of loads)
  int want = (2 * num_sms() + n - 1) / n;
  int maxc = hw / (p.rows * 4);
  if (maxc < 1) maxc = 1;
  p.nchunks = want < maxc ? want : maxc;
  return p;
}

namespace {

template <typename T>
__device__ __forceinline__ const T* cat_ptr(const T* p0, int c0, const T* p1, int c1, size_t pix, int ch) {
  return ch < c0 ? p0 + pix * c0 + ch : p1 + pix * c1 + (ch - c0);
}

// dynamic shared memory layout of every kernel here: [2C] channel sums | [2G] group values | reduction scratch
struct Smem {
  float* cs;     // [2][C]
  float* grp;    // [2][G]
  float* red;    // [rows][k][C]
  __device__ Smem(float* base, int C, int G) : cs(base), grp(base + 2 * C), red(base + 2 * C + 2 * G) {}
};
size_t smem_bytes(int C, int G, int rows, int k) {
  return ((size_t)2 * C + 2 * G + (rows > 1 ? (size_t)rows * k * C : 0)) * sizeof(float);
}

__device__ __forceinline__ int tid_() { return threadIdx.y * blockDim.x + threadIdx.x; }
__device__ __forceinline__ int nthr_() { return blockDim.x * blockDim.y; }

// grp[g] = mean, grp[G+g] = rstd of group g of image n, from the channel stats of the two sources
// PIV (fp32 tensors): the sums are of (x - pivot_c), pivot_c = x[n, pixel 0, c] (chan_stats_k); they are turned into
// plain per-channel moments in ACC = double here, where the cancellation is harmless.
template <typename ACC, bool PIV, typename T>
__device__ __forceinline__ void group_mean_rstd(const float* __restrict__ cst0, int c0, const float* __restrict__ cst1,
                                                int c1, int n, int hw, int G, float eps, Smem& s, const T* __restrict__ p0,
                                                const T* __restrict__ p1) {
  const int C = c0 + c1, tid = tid_(), nthr = nthr_(), cpg = C / G;
  for (int i0 = tid; i0 < 2 * C; i0 += 4 * nthr) {      // 4 independent loads per thread in flight: one L2 round trip
    float v[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int i = i0 + u * nthr;
      if (i < 2 * C) {
        const int which = i >= C ? 1 : 0, c = i - which * C;
        v[u] = c < c0 ? cst0[((size_t)n * 2 + which) * c0 + c] : cst1[((size_t)n * 2 + which) * c1 + (c - c0)];
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u)
      if (i0 + u * nthr < 2 * C) s.cs[i0 + u * nthr] = v[u];
  }
  __syncthreads();
  // combined in ACC (R22: double on the fp32 debug path; fp32 for bf16 tensors, where fp64 division / sqrt cost
  // microseconds per kernel); 4 threads per group when the CTA has that many whole warps
  const bool quad = nthr >= ((4 * G + 31) & ~31);
  const int L = quad ? 4 : 1;
  for (int g0 = 0; g0 < G; g0 += quad ? G : nthr) {
    const int g = g0 + tid / L, l = tid % L;
    ACC a = 0, b = 0;
    if (g < G)
      for (int c = g * cpg + l; c < (g + 1) * cpg; c += L) {
        ACC s1 = (ACC)s.cs[c], s2 = (ACC)s.cs[C + c];
        if (PIV) {      // sum x = s1 + hw p; sum x^2 = s2 + 2 p s1 + hw p^2
          const ACC pv = (ACC)to_f(c < c0 ? p0[(size_t)n * hw * c0 + c] : p1[(size_t)n * hw * c1 + (c - c0)]);
          s2 += (ACC)2 * pv * s1 + (ACC)hw * pv * pv;
          s1 += (ACC)hw * pv;
        }
        a += s1; b += s2;
      }
    if (quad && tid < ((4 * G + 31) & ~31)) {
      a += __shfl_xor_sync(0xffffffffu, a, 1); b += __shfl_xor_sync(0xffffffffu, b, 1);
      a += __shfl_xor_sync(0xffffffffu, a, 2); b += __shfl_xor_sync(0xffffffffu, b, 2);
    }
    if (g < G && l == 0) {
      const ACC m = (ACC)cpg * (ACC)hw, mu = a / m;
      ACC var = b / m - mu * mu;
      if (var < 0) var = 0;
      s.grp[g] = (float)mu;
      s.grp[G + g] = (float)((ACC)1 / sqrt(var + (ACC)eps));
    }
  }
  __syncthreads();
}

// backward kernels: mean / rstd [n][2G] as the forward apply saved them (no statistics prologue)
__device__ __forceinline__ void load_mean_rstd(const float* __restrict__ mr, int n, int G, Smem& s) {
  for (int i = tid_(); i < 2 * G; i += nthr_()) s.grp[i] = mr[(size_t)n * 2 * G + i];
  __syncthreads();
}

// per-thread normalisation coefficients of V consecutive channels: y = x sc + sh, xhat = x rr - mr
template <typename T, int V>
__device__ __forceinline__ void gn_coefs(const Smem& s, int G, int cpg, const float (&gav)[V], const float (&bev)[V],
                                         int ch, float (&sc)[V], float (&sh)[V], float (&rr)[V], float (&mr)[V]) {
  int g = ch / cpg, rem = ch - g * cpg;          // one division; the V channels then walk the groups
#pragma unroll
  for (int i = 0; i < V; ++i) {
    const float mu = s.grp[g], r = s.grp[G + g];
    const float ga = gav[i], be = bev[i];
    rr[i] = r; mr[i] = mu * r;
    sc[i] = r * ga; sh[i] = be - mr[i] * ga;
    if (++rem == cpg) { rem = 0; ++g; }
  }
}

// sum the per-thread partials v[2][V] over the rows of the CTA and add them into dst[2][C] (global, one atomic
// per channel per CTA)
template <int V>
__device__ __forceinline__ void reduce_rows_atomic(float (&v)[2][V], int C, Smem& s, float* dst) {
  const int rows = blockDim.y, ch = threadIdx.x * V;
  if (rows == 1) {
#pragma unroll
    for (int k = 0; k < 2; ++k)
#pragma unroll
      for (int i = 0; i < V; ++i) atomicAdd(dst + k * C + ch + i, v[k][i]);
    return;
  }
#pragma unroll
  for (int k = 0; k < 2; ++k)
#pragma unroll
    for (int i = 0; i < V; ++i) s.red[((size_t)threadIdx.y * 2 + k) * C + ch + i] = v[k][i];
  __syncthreads();
  for (int j = tid_(); j < 2 * C; j += nthr_()) {
    float t = 0.f;
    for (int r = 0; r < rows; ++r) t += s.red[(size_t)r * 2 * C + j];
    atomicAdd(dst + j, t);
  }
}


// ---- shared-memory ring fed by bulk asynchronous copies -----------------------------------------------------
constexpr int RS = 3;        // ring stages
constexpr int MAXS = 4;      // input streams per kernel
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(sm100::smem_u32(smem_dst)), "l"(gsrc), "r"(bytes), "r"(sm100::smem_u32(bar)) : "memory");
}
struct Ring {
  uint64_t* full;            // [RS]
  uint8_t* buf;
  int ns = 0;
  const char* g[MAXS]; int ppb[MAXS]; int soff[MAXS];    // global base (pixel 0 of this image), bytes per pixel, offset in a stage
  int stage_bytes, P, pb, pe, nch;
  // stream i of every stage holds P pixels of `bytes_per_pixel` bytes
  __device__ __forceinline__ int add(const void* base, int bytes_per_pixel) {
    g[ns] = (const char*)base; ppb[ns] = bytes_per_pixel; soff[ns] = ns ? soff[ns - 1] + P * ppb[ns - 1] : 0;
    return ns++;
  }
  __device__ __forceinline__ void issue(int c) {            // one thread
    const int s = c % RS, p0 = pb + c * P, np = min(P, pe - p0);
    uint32_t bytes = 0;
    for (int i = 0; i < ns; ++i) bytes += (uint32_t)np * ppb[i];
    sm100::mbar_expect_tx(&full[s], bytes);
    for (int i = 0; i < ns; ++i)
      bulk_g2s(buf + (size_t)s * stage_bytes + soff[i], g[i] + (size_t)p0 * ppb[i], (uint32_t)np * ppb[i], &full[s]);
  }
  __device__ __forceinline__ void start(int tid) {          // whole CTA; barriers are initialised here
    if (tid == 0) {
      for (int i = 0; i < RS; ++i) sm100::mbar_init(&full[i], 1);
      sm100::fence_barrier_init();
      for (int c = 0; c < RS && c < nch; ++c) issue(c);
    }
    __syncthreads();
  }
  __device__ __forceinline__ const uint8_t* wait(int c) {
    sm100::mbar_wait(&full[c % RS], (c / RS) & 1);
    return buf + (size_t)(c % RS) * stage_bytes;
  }
  __device__ __forceinline__ void release(int c, int tid) { // whole CTA: everyone is done reading stage c % RS
    __syncthreads();
    if (tid == 0 && c + RS < nch) issue(c + RS);
  }
};
// load Vec<T>::N consecutive elements from shared memory (generic pointer) into floats
template <typename T> __device__ __forceinline__ void lds(const uint8_t* p, float (&o)[Vec<T>::N]) {
  ldv(reinterpret_cast<const T*>(p), o);
}

// ------------------------------------------------------------------------------ channel stats of one tensor
template <typename T>
__global__ void __launch_bounds__(512, 2) chan_stats_k(const T* __restrict__ x, int C, int hw, float* __restrict__ cst,
                                                        T* __restrict__ copy) {     // copy (nullable): also copy x there
  constexpr int V = Vec<T>::N;
  extern __shared__ float sm_[];
  Smem s(sm_, C, 0);
  const int n = blockIdx.y, nchunks = gridDim.x, rows = blockDim.y;
  const int ppc = (hw + nchunks - 1) / nchunks;
  const int pb = blockIdx.x * ppc, pe = min(hw, pb + ppc);
  const int ch = threadIdx.x * V;
  float v[2][V], piv[V];
#pragma unroll
  for (int i = 0; i < V; ++i) v[0][i] = v[1][i] = 0.f;
  // fp32 path (R22): sums of (x - pivot), pivot = the channel's value at pixel 0 of the image, so that a channel mean far
  // from zero does not cancel in E[x^2] - E[x]^2; the consumer (group_mean_rstd) reads the same pivot from x itself.
  // bf16 tensors (statistics also come from conv epilogues, which see one tile each) keep plain sums.
  if (sizeof(T) == 4) ldv(x + (size_t)n * hw * C + ch, piv);
  else {
#pragma unroll
    for (int i = 0; i < V; ++i) piv[i] = 0.f;
  }
  for (int p = pb + threadIdx.y; p < pe; p += 4 * rows) {
    float t[4][V];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      if (p + u * rows < pe) {
        const size_t off = ((size_t)n * hw + p + u * rows) * C + ch;
        const uint4 raw = *reinterpret_cast<const uint4*>(x + off);       // 16 bytes = V elements
        if (copy) *reinterpret_cast<uint4*>(copy + off) = raw;
        unpack(raw, t[u]);
#pragma unroll
        for (int i = 0; i < V; ++i) t[u][i] -= piv[i];
      } else {
#pragma unroll
        for (int i = 0; i < V; ++i) t[u][i] = 0.f;
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int i = 0; i < V; ++i) { v[0][i] += t[u][i]; v[1][i] = fmaf(t[u][i], t[u][i], v[1][i]); }
  }
  reduce_rows_atomic<V>(v, C, s, cst + (size_t)n * 2 * C);
}

// SiLU pieces: sigmoid = 1 / (1 + 2^(-y log2 e)): one MUFU.EX2 and one MUFU.RCP per element.  (The single-MUFU
// tanh.approx form, sigmoid = 0.5 tanh(y/2) + 0.5, was measured and rejected: its 2^-11 relative error is a smooth
// function of y, so it does not average out in the bias / gamma / beta sums and pushed small-tensor gradients past
// the 2e-2 bar.)
template <typename T> __device__ __forceinline__ float sigmoid_t(float y) { return sigmoidf_(y); }
template <typename T> __device__ __forceinline__ float silu_t(float y) { return y * sigmoid_t<T>(y); }
template <typename T> __device__ __forceinline__ float silu_grad_t(float y) {
  const float s = sigmoid_t<T>(y);
  return fmaf(y * s, 1.0f - s, s);
}

// dynamic smem: [prologue floats (Smem)] | pad to 128 | ring.  `pro_floats` = size of the first part.
__device__ __forceinline__ uint8_t* ring_base(float* sm, int pro_floats) {
  return reinterpret_cast<uint8_t*>(sm) + (((size_t)pro_floats * 4 + 127) & ~(size_t)127);
}

// ------------------------------------------------------------------------------ forward apply (one pass)
// ACT (here and in the backward kernels): 1 = GroupNorm + SiLU, 0 = plain GroupNorm (attention blocks); a template parameter
// because the pixel loops are bound by instruction issue
template <typename T, int ACT>
__global__ void __launch_bounds__(512, 2)
gn_apply_k(const T* __restrict__ p0, int c0, const T* __restrict__ p1, int c1, int hw, int G, float eps,
           const T* __restrict__ gamma, const T* __restrict__ beta, const float* __restrict__ cst0,
           const float* __restrict__ cst1, float* __restrict__ mr_out, T* __restrict__ out, int P, int stage_bytes,
           int pro_floats) {
  constexpr int V = Vec<T>::N;
  extern __shared__ float sm_[];
  __shared__ uint64_t full[RS];
  const int C = c0 + c1, n = blockIdx.y, nchunks = gridDim.x, rows = blockDim.y, tid = tid_();
  Smem s(sm_, C, G);
  const int ppc = (hw + nchunks - 1) / nchunks;
  const int ch = threadIdx.x * V;
  Ring r;
  r.full = full; r.buf = ring_base(sm_, pro_floats); r.P = P; r.stage_bytes = stage_bytes;
  r.pb = blockIdx.x * ppc; r.pe = min(hw, r.pb + ppc); r.nch = r.pe > r.pb ? (r.pe - r.pb + P - 1) / P : 0;
  const int i0 = r.add(p0 + (size_t)n * hw * c0, c0 * (int)sizeof(T));
  const int i1 = c1 ? r.add(p1 + (size_t)n * hw * c1, c1 * (int)sizeof(T)) : i0;
  float gav[V], bev[V];                 // parameters: loaded before the dependency wait
#pragma unroll
  for (int i = 0; i < V; ++i) { gav[i] = to_f(gamma[ch + i]); bev[i] = to_f(beta[ch + i]); }
  pdl_wait();
  pdl_launch_dependents();
  r.start(tid);
  group_mean_rstd<typename std::conditional<sizeof(T) == 4, double, float>::type, sizeof(T) == 4, T>(cst0, c0, cst1, c1, n, hw,
                                                                                                     G, eps, s, p0, p1);
  if (blockIdx.x == 0)        // mean / rstd for the backward kernels of this site
    for (int i = tid; i < 2 * G; i += nthr_()) mr_out[(size_t)n * 2 * G + i] = s.grp[i];
  float sc[V], sh[V], rr[V], mr[V];
  gn_coefs<T, V>(s, G, C / G, gav, bev, ch, sc, sh, rr, mr);
  const bool lo = ch < c0;
  const int xoff = lo ? r.soff[i0] + ch * (int)sizeof(T) : r.soff[i1] + (ch - c0) * (int)sizeof(T);
  const int xpp = lo ? r.ppb[i0] : r.ppb[i1];
  for (int c = 0; c < r.nch; ++c) {
    const uint8_t* st = r.wait(c);
    const int pbase = r.pb + c * P, np = min(P, r.pe - pbase);
    for (int pl = threadIdx.y; pl < np; pl += 2 * rows) {      // two independent pixels per iteration (ILP)
      float v[2][V];
      const bool two = pl + rows < np;
      lds<T>(st + xoff + pl * xpp, v[0]);
      if (two) lds<T>(st + xoff + (pl + rows) * xpp, v[1]);
#pragma unroll
      for (int i = 0; i < V; ++i) {
        const float y0 = fmaf(v[0][i], sc[i], sh[i]), y1 = fmaf(v[1][i], sc[i], sh[i]);
        v[0][i] = ACT ? silu_t<T>(y0) : y0;          // act == 0: plain GroupNorm (attention blocks)
        v[1][i] = ACT ? silu_t<T>(y1) : y1;
      }
      stv(out + ((size_t)n * hw + pbase + pl) * C + ch, v[0]);
      if (two) stv(out + ((size_t)n * hw + pbase + pl + rows) * C + ch, v[1]);
    }
    r.release(c, tid);
  }
}

// ------------------------------------------------------------------------------ backward: reduction pass
// bst[n][0][c] += sum_pix g_y, bst[n][1][c] += sum_pix g_y xhat
template <typename T, int ACT>
__global__ void __launch_bounds__(512, 1)
gn_bwd_stats_k(const T* __restrict__ ga, const T* __restrict__ p0, int c0, const T* __restrict__ p1, int c1, int hw,
               int G, float eps, const T* __restrict__ gamma, const T* __restrict__ beta,
               const float* __restrict__ mrp, float* __restrict__ bst, int P, int stage_bytes, int pro_floats) {
  constexpr int V = Vec<T>::N;
  extern __shared__ float sm_[];
  __shared__ uint64_t full[RS];
  const int C = c0 + c1, n = blockIdx.y, nchunks = gridDim.x, rows = blockDim.y, tid = tid_();
  Smem s(sm_, C, G);
  const int ppc = (hw + nchunks - 1) / nchunks;
  const int ch = threadIdx.x * V;
  Ring r;
  r.full = full; r.buf = ring_base(sm_, pro_floats); r.P = P; r.stage_bytes = stage_bytes;
  r.pb = blockIdx.x * ppc; r.pe = min(hw, r.pb + ppc); r.nch = r.pe > r.pb ? (r.pe - r.pb + P - 1) / P : 0;
  const int i0 = r.add(p0 + (size_t)n * hw * c0, c0 * (int)sizeof(T));
  const int i1 = c1 ? r.add(p1 + (size_t)n * hw * c1, c1 * (int)sizeof(T)) : i0;
  const int ig = r.add(ga + (size_t)n * hw * C, C * (int)sizeof(T));
  float gav[V], bev[V];                 // parameters: loaded before the dependency wait
#pragma unroll
  for (int i = 0; i < V; ++i) { gav[i] = to_f(gamma[ch + i]); bev[i] = to_f(beta[ch + i]); }
  pdl_wait();
  pdl_launch_dependents();
  r.start(tid);
  load_mean_rstd(mrp, n, G, s);
  float sc[V], sh[V], rr[V], mr[V], v[2][V];
  gn_coefs<T, V>(s, G, C / G, gav, bev, ch, sc, sh, rr, mr);
#pragma unroll
  for (int i = 0; i < V; ++i) v[0][i] = v[1][i] = 0.f;
  const bool lo = ch < c0;
  const int xoff = lo ? r.soff[i0] + ch * (int)sizeof(T) : r.soff[i1] + (ch - c0) * (int)sizeof(T);
  const int xpp = lo ? r.ppb[i0] : r.ppb[i1];
  const int goff = r.soff[ig] + ch * (int)sizeof(T), gpp = r.ppb[ig];
  for (int c = 0; c < r.nch; ++c) {
    const uint8_t* st = r.wait(c);
    const int np = min(P, r.pe - (r.pb + c * P));
    for (int pl = threadIdx.y; pl < np; pl += rows) {
      float x[V], g[V];
      lds<T>(st + xoff + pl * xpp, x);
      lds<T>(st + goff + pl * gpp, g);
#pragma unroll
      for (int i = 0; i < V; ++i) {
        const float gy = ACT ? g[i] * silu_grad_t<T>(fmaf(x[i], sc[i], sh[i])) : g[i];
        v[0][i] += gy;
        v[1][i] = fmaf(gy, fmaf(x[i], rr[i], -mr[i]), v[1][i]);
      }
    }
    r.release(c, tid);
  }
  reduce_rows_atomic<V>(v, C, s, bst + (size_t)n * 2 * C);
}

// ------------------------------------------------------------------------------ backward: apply pass
// g_x = r (gamma g_y - A - xhat B) [+ add]; channels [0,dc0) -> dst0, the rest -> dst1 (skip gradient,
// PAPER.md:L91); acc: += instead of =.  cs0/cs1: per-(image, channel) sums of what this launch ADDS to
// dst0/dst1 (before bf16 rounding), accumulated.  dgamma/dbeta: += sum_n bst (CTA chunk 0 of each image).
template <typename T, int ACT>
__global__ void __launch_bounds__(512, 1)
gn_bwd_apply_k(const T* __restrict__ ga, const T* __restrict__ p0, int c0, const T* __restrict__ p1, int c1, int hw,
               int G, float eps, const T* __restrict__ gamma, const T* __restrict__ beta,
               const float* __restrict__ mrp, const float* __restrict__ bst, float* dgamma, float* dbeta, const T* __restrict__ add, T* dst0, int dc0, int acc0, T* dst1, int acc1,
               float* cs0, float* cs1, int P, int stage_bytes, int pro_floats) {
  constexpr int V = Vec<T>::N;
  extern __shared__ float sm_[];
  __shared__ uint64_t full[RS];
  const int C = c0 + c1, n = blockIdx.y, nchunks = gridDim.x, rows = blockDim.y, cpg = C / G;
  Smem s(sm_, C, G);
  const int ppc = (hw + nchunks - 1) / nchunks;
  const int ch = threadIdx.x * V, tid = tid_(), nthr = nthr_();
  Ring r;
  r.full = full; r.buf = ring_base(sm_, pro_floats); r.P = P; r.stage_bytes = stage_bytes;
  r.pb = blockIdx.x * ppc; r.pe = min(hw, r.pb + ppc); r.nch = r.pe > r.pb ? (r.pe - r.pb + P - 1) / P : 0;
  const int i0 = r.add(p0 + (size_t)n * hw * c0, c0 * (int)sizeof(T));
  const int i1 = c1 ? r.add(p1 + (size_t)n * hw * c1, c1 * (int)sizeof(T)) : i0;
  const int ig = r.add(ga + (size_t)n * hw * C, C * (int)sizeof(T));
  const int ie = add ? r.add(add + (size_t)n * hw * C, C * (int)sizeof(T)) : ig;
  float gav[V], bev[V];                 // parameters: loaded before the dependency wait
#pragma unroll
  for (int i = 0; i < V; ++i) { gav[i] = to_f(gamma[ch + i]); bev[i] = to_f(beta[ch + i]); }
  pdl_wait();
  pdl_launch_dependents();
  r.start(tid);
  load_mean_rstd(mrp, n, G, s);
  float sc[V], sh[V], rr[V], mr[V], k2[V], k3[V];
  gn_coefs<T, V>(s, G, cpg, gav, bev, ch, sc, sh, rr, mr);
  // group sums A m = sum_c gamma_c S1[c], B m = sum_c gamma_c S2[c]  (s.cs is free again: reuse it for S1|S2)
  __syncthreads();
  for (int i = tid; i < 2 * C; i += nthr) {
    const float t = bst[(size_t)n * 2 * C + i];
    s.cs[i] = t;
    if (blockIdx.x == 0) {
      if (i < C) atomicAdd(dbeta + i, t); else atomicAdd(dgamma + (i - C), t);
    }
  }
  __syncthreads();
  {   // everyone has read s.grp (mean, rstd) through gn_coefs and synchronised since: overwrite it with A/m, B/m
    const bool quad = nthr >= ((4 * G + 31) & ~31);
    const int L = quad ? 4 : 1;
    const float inv = 1.0f / ((float)cpg * (float)hw);
    for (int g0 = 0; g0 < G; g0 += quad ? G : nthr) {
      const int g = g0 + tid / L, l = tid % L;
      float a = 0.f, b = 0.f;
      if (g < G)
        for (int c = g * cpg + l; c < (g + 1) * cpg; c += L) {
          const float ga_ = to_f(gamma[c]);
          a = fmaf(ga_, s.cs[c], a); b = fmaf(ga_, s.cs[C + c], b);
        }
      if (quad && tid < ((4 * G + 31) & ~31)) {
        a += __shfl_xor_sync(0xffffffffu, a, 1); b += __shfl_xor_sync(0xffffffffu, b, 1);
        a += __shfl_xor_sync(0xffffffffu, a, 2); b += __shfl_xor_sync(0xffffffffu, b, 2);
      }
      if (g < G && l == 0) { s.grp[g] = a * inv; s.grp[G + g] = b * inv; }
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < V; ++i) {
    const int g = (ch + i) / cpg;
    k2[i] = s.grp[g] * rr[i];
    k3[i] = s.grp[G + g] * rr[i];
  }
  const bool first = ch < dc0;
  T* dst = first ? dst0 : dst1;
  const int dC = first ? dc0 : C - dc0, dch = first ? ch : ch - dc0;
  const int acc = first ? acc0 : acc1;
  float sum[V];
#pragma unroll
  for (int i = 0; i < V; ++i) sum[i] = 0.f;
  const bool lo = ch < c0;
  const int xoff = lo ? r.soff[i0] + ch * (int)sizeof(T) : r.soff[i1] + (ch - c0) * (int)sizeof(T);
  const int xpp = lo ? r.ppb[i0] : r.ppb[i1];
  const int goff = r.soff[ig] + ch * (int)sizeof(T), eoff = r.soff[ie] + ch * (int)sizeof(T), gpp = C * (int)sizeof(T);
  for (int c = 0; c < r.nch; ++c) {
    const uint8_t* st = r.wait(c);
    const int pbase = r.pb + c * P, np = min(P, r.pe - pbase);
    for (int pl = threadIdx.y; pl < np; pl += rows) {
      const size_t pix = (size_t)n * hw + pbase + pl;
      float x[V], g[V], e[V], f[V], o[V];
      if (acc) ldv(dst + pix * dC + dch, f);          // the only non-streamed input (second writer of a gradient)
      lds<T>(st + xoff + pl * xpp, x);
      lds<T>(st + goff + pl * gpp, g);
      if (add) lds<T>(st + eoff + pl * gpp, e);
#pragma unroll
      for (int i = 0; i < V; ++i) {
        const float gy = ACT ? g[i] * silu_grad_t<T>(fmaf(x[i], sc[i], sh[i])) : g[i];
        const float xh = fmaf(x[i], rr[i], -mr[i]);
        o[i] = sc[i] * gy - k2[i] - xh * k3[i];
        if (add) o[i] += e[i];
        sum[i] += o[i];
        if (acc) o[i] += f[i];
      }
      stv(dst + pix * dC + dch, o);
    }
    r.release(c, tid);
  }
  if (cs0 || cs1) {      // channels below dc0 -> cs0[n][dc0], the rest -> cs1[n][C - dc0]
    if (rows == 1) {
#pragma unroll
      for (int i = 0; i < V; ++i) {
        const int c = ch + i;
        if (c < dc0) { if (cs0) atomicAdd(cs0 + (size_t)n * dc0 + c, sum[i]); }
        else if (cs1) atomicAdd(cs1 + (size_t)n * (C - dc0) + (c - dc0), sum[i]);
      }
    } else {
#pragma unroll
      for (int i = 0; i < V; ++i) s.red[(size_t)threadIdx.y * C + ch + i] = sum[i];
      __syncthreads();
      for (int c = tid; c < C; c += nthr) {
        float t = 0.f;
        for (int r = 0; r < rows; ++r) t += s.red[(size_t)r * C + c];
        if (c < dc0) { if (cs0) atomicAdd(cs0 + (size_t)n * dc0 + c, t); }
        else if (cs1) atomicAdd(cs1 + (size_t)n * (C - dc0) + (c - dc0), t);
      }
    }
  }
}

}  // namespace

// ------------------------------------------------------------------------------ host launchers
int chan_stats(int dt, const void* x, int n, int hw, int c, float* cst, cudaStream_t st, void* copy) {
  const RowPlan pl = row_plan(dt, hw, c, n, 512);
  dim3 grid(pl.nchunks, n), block(pl.tpr, pl.rows);
  const size_t sm = smem_bytes(c, 0, pl.rows, 2);
  if (dt == DT_F32) chan_stats_k<float><<<grid, block, sm, st>>>((const float*)x, c, hw, cst, (float*)copy);
  else chan_stats_k<bf16><<<grid, block, sm, st>>>((const bf16*)x, c, hw, cst, (bf16*)copy);
  return 1;
}

// launch geometry of the streaming kernels: one CTA per SM over the whole grid, <= 512 threads; P pixels per ring
// stage so that a stage is <= 56 KB (3 stages + prologue stay under the 227 KB of shared memory)
struct StreamPlan { dim3 grid, block; int P, stage_bytes, pro_floats; size_t smem; };
static StreamPlan stream_plan(int dt, int n, int hw, int C, int G, int red_k, int bytes_per_pixel, int ctas_per_sm = 1) {
  StreamPlan sp;
  const int vec = dt == DT_F32 ? 4 : 8;
  const int tpr = C / vec;
  int rows = tpr >= 512 ? 1 : 512 / tpr;
  if (rows > hw) rows = hw;
  int ppt = (56 * 1024 / ctas_per_sm) / (rows * bytes_per_pixel);
  if (ppt < 1) ppt = 1;
  if (ppt > 8) ppt = 8;
  sp.P = rows * ppt;
  sp.stage_bytes = (sp.P * bytes_per_pixel + 127) & ~127;
  int nchunks = (ctas_per_sm * num_sms() + n - 1) / n;
  const int maxc = (hw + rows - 1) / rows;        // at least one pixel per thread row
  if (nchunks > maxc) nchunks = maxc;
  if (nchunks < 1) nchunks = 1;
  sp.grid = dim3(nchunks, n); sp.block = dim3(tpr, rows);
  sp.pro_floats = 2 * C + 2 * G + (rows > 1 ? rows * red_k * C : 0);
  sp.smem = (((size_t)sp.pro_floats * 4 + 127) & ~(size_t)127) + (size_t)RS * sp.stage_bytes;
  return sp;
}
template <typename K> static void allow_big_smem(K kernel) {
  cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 1024);
}

template <typename T, int ACT>
static void gn_fwd_t(Cat x, int n, int hw, int groups, float eps, const void* gamma, const void* beta, const float* cst0,
                     const float* cst1, float* mr_out, void* a_out, cudaStream_t st) {
  const int C = x.c();
  const StreamPlan sp = stream_plan(sizeof(T) == 4 ? DT_F32 : DT_BF16, n, hw, C, groups, 0, C * (int)sizeof(T), 2);
  static bool attr = false;
  if (!attr) { allow_big_smem(gn_apply_k<T, ACT>); attr = true; }
  launch_pdl(gn_apply_k<T, ACT>, sp.grid, sp.block, sp.smem, st, (const T*)x.p0, x.c0, (const T*)x.p1, x.c1, hw, groups, eps,
             (const T*)gamma, (const T*)beta, cst0, cst1, mr_out, (T*)a_out, sp.P, sp.stage_bytes, sp.pro_floats);
}

int gn_silu_fwd(int dt, Cat x, int n, int hw, int groups, float eps, const void* gamma, const void* beta,
                const float* cst0, const float* cst1, float* mr_out, void* a_out, cudaStream_t st, int act) {
  if (dt == DT_F32) {
    if (act) gn_fwd_t<float, 1>(x, n, hw, groups, eps, gamma, beta, cst0, cst1, mr_out, a_out, st);
    else gn_fwd_t<float, 0>(x, n, hw, groups, eps, gamma, beta, cst0, cst1, mr_out, a_out, st);
  } else {
    if (act) gn_fwd_t<bf16, 1>(x, n, hw, groups, eps, gamma, beta, cst0, cst1, mr_out, a_out, st);
    else gn_fwd_t<bf16, 0>(x, n, hw, groups, eps, gamma, beta, cst0, cst1, mr_out, a_out, st);
  }
  return 1;
}

template <typename T, int ACT>
static int gn_bwd_t(const void* g_a, Cat x, int n, int hw, int groups, float eps, const void* gamma, const void* beta,
                    const float* mr, float* bst, const void* add, void* dst0, int dc0, int acc0,
                    void* dst1, int acc1, float* dgamma, float* dbeta, float* cs0, float* cs1, cudaStream_t st,
                    bool allow_fused, bool fwd_data_ready) {
  const int C = x.c();
  const int dt = sizeof(T) == 4 ? DT_F32 : DT_BF16;
  if (dt == DT_BF16 && allow_fused) {        // one pass with the tensors resident in shared memory where the shape allows (norm_fused.cu)
    const int r = gn_bwd_fused(g_a, x, n, hw, groups, gamma, beta, mr, add, dst0, dc0, acc0, dst1, acc1, dgamma, dbeta,
                               cs0, cs1, st, fwd_data_ready, ACT);
    if (r > 0) return r;
  }
  static bool attr = false;
  if (!attr) { allow_big_smem(gn_bwd_stats_k<T, ACT>); allow_big_smem(gn_bwd_apply_k<T, ACT>); attr = true; }
  const StreamPlan s1 = stream_plan(dt, n, hw, C, groups, 2, 2 * C * (int)sizeof(T));
  launch_pdl(gn_bwd_stats_k<T, ACT>, s1.grid, s1.block, s1.smem, st, (const T*)g_a, (const T*)x.p0, x.c0, (const T*)x.p1,
             x.c1, hw, groups, eps, (const T*)gamma, (const T*)beta, mr, bst, s1.P, s1.stage_bytes, s1.pro_floats);
  const StreamPlan s2 = stream_plan(dt, n, hw, C, groups, 1, (add ? 3 : 2) * C * (int)sizeof(T));
  launch_pdl(gn_bwd_apply_k<T, ACT>, s2.grid, s2.block, s2.smem, st, (const T*)g_a, (const T*)x.p0, x.c0, (const T*)x.p1,
             x.c1, hw, groups, eps, (const T*)gamma, (const T*)beta, mr, (const float*)bst, dgamma, dbeta,
             (const T*)add, (T*)dst0, dc0, acc0, (T*)dst1, acc1, cs0, cs1, s2.P, s2.stage_bytes, s2.pro_floats);
  return 2;
}

int gn_silu_bwd(int dt, const void* g_a, Cat x, int n, int hw, int groups, float eps, const void* gamma,
                const void* beta, const float* mr, float* bst, const void* add, void* dst0,
                int dc0, int acc0, void* dst1, int acc1, float* dgamma, float* dbeta, float* cs0, float* cs1,
                cudaStream_t st, bool allow_fused, bool fwd_data_ready, int act) {
#define PULSE_GN_BWD(T, A, FUSED)                                                                                       \
  gn_bwd_t<T, A>(g_a, x, n, hw, groups, eps, gamma, beta, mr, bst, add, dst0, dc0, acc0, dst1, acc1, dgamma, dbeta, cs0, \
                 cs1, st, FUSED, fwd_data_ready)
  if (dt == DT_F32) return act ? PULSE_GN_BWD(float, 1, false) : PULSE_GN_BWD(float, 0, false);
  return act ? PULSE_GN_BWD(bf16, 1, allow_fused) : PULSE_GN_BWD(bf16, 0, allow_fused);
#undef PULSE_GN_BWD
}

}  // namespace pulse

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
#include "common.cuh"
#include "kernels.h"

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
__device__ __forceinline__ void group_mean_rstd(const float* __restrict__ cst0, int c0, const float* __restrict__ cst1,
                                                int c1, int n, int hw, int G, float eps, Smem& s) {
  const int C = c0 + c1, tid = tid_(), nthr = nthr_(), cpg = C / G;
  for (int i = tid; i < 2 * C; i += nthr) {
    const int which = i / C, c = i - which * C;
    s.cs[i] = c < c0 ? cst0[((size_t)n * 2 + which) * c0 + c] : cst1[((size_t)n * 2 + which) * c1 + (c - c0)];
  }
  __syncthreads();
  // combined in double (R22); 4 threads per group when the CTA has that many whole warps
  const bool quad = nthr >= ((4 * G + 31) & ~31);
  const int L = quad ? 4 : 1;
  for (int g0 = 0; g0 < G; g0 += quad ? G : nthr) {
    const int g = g0 + tid / L, l = tid % L;
    double a = 0.0, b = 0.0;
    if (g < G)
      for (int c = g * cpg + l; c < (g + 1) * cpg; c += L) { a += (double)s.cs[c]; b += (double)s.cs[C + c]; }
    if (quad && tid < ((4 * G + 31) & ~31)) {
      a += __shfl_xor_sync(0xffffffffu, a, 1); b += __shfl_xor_sync(0xffffffffu, b, 1);
      a += __shfl_xor_sync(0xffffffffu, a, 2); b += __shfl_xor_sync(0xffffffffu, b, 2);
    }
    if (g < G && l == 0) {
      const double m = (double)cpg * hw, mu = a / m;
      double var = b / m - mu * mu;
      if (var < 0.0) var = 0.0;
      s.grp[g] = (float)mu;
      s.grp[G + g] = (float)(1.0 / sqrt(var + (double)eps));
    }
  }
  __syncthreads();
}

// per-thread normalisation coefficients of V consecutive channels: y = x sc + sh, xhat = x rr - mr
template <typename T, int V>
__device__ __forceinline__ void gn_coefs(const Smem& s, int G, int cpg, const T* __restrict__ gamma,
                                         const T* __restrict__ beta, int ch, float (&sc)[V], float (&sh)[V],
                                         float (&rr)[V], float (&mr)[V]) {
#pragma unroll
  for (int i = 0; i < V; ++i) {
    const int g = (ch + i) / cpg;
    const float mu = s.grp[g], r = s.grp[G + g];
    const float ga = to_f(gamma[ch + i]), be = to_f(beta[ch + i]);
    rr[i] = r; mr[i] = mu * r;
    sc[i] = r * ga; sh[i] = be - mr[i] * ga;
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

// ------------------------------------------------------------------------------ channel stats of one tensor
template <typename T>
__global__ void __launch_bounds__(512, 2) chan_stats_k(const T* __restrict__ x, int C, int hw, float* __restrict__ cst) {
  constexpr int V = Vec<T>::N;
  extern __shared__ float sm_[];
  Smem s(sm_, C, 0);
  const int n = blockIdx.y, nchunks = gridDim.x, rows = blockDim.y;
  const int ppc = (hw + nchunks - 1) / nchunks;
  const int pb = blockIdx.x * ppc, pe = min(hw, pb + ppc);
  const int ch = threadIdx.x * V;
  float v[2][V];
#pragma unroll
  for (int i = 0; i < V; ++i) v[0][i] = v[1][i] = 0.f;
  for (int p = pb + threadIdx.y; p < pe; p += 4 * rows) {
    float t[4][V];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      if (p + u * rows < pe) ldv(x + ((size_t)n * hw + p + u * rows) * C + ch, t[u]);
      else {
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

// ------------------------------------------------------------------------------ forward apply (one pass)
template <typename T>
__global__ void __launch_bounds__(512, 2)
gn_apply_k(const T* __restrict__ p0, int c0, const T* __restrict__ p1, int c1, int hw, int G, float eps,
           const T* __restrict__ gamma, const T* __restrict__ beta, const float* __restrict__ cst0,
           const float* __restrict__ cst1, T* __restrict__ out) {
  constexpr int V = Vec<T>::N;
  extern __shared__ float sm_[];
  const int C = c0 + c1, n = blockIdx.y, nchunks = gridDim.x, rows = blockDim.y;
  Smem s(sm_, C, G);
  const int ppc = (hw + nchunks - 1) / nchunks;
  const int pb = blockIdx.x * ppc, pe = min(hw, pb + ppc);
  const int ch = threadIdx.x * V;
  group_mean_rstd(cst0, c0, cst1, c1, n, hw, G, eps, s);
  float sc[V], sh[V], rr[V], mr[V];
  gn_coefs<T, V>(s, G, C / G, gamma, beta, ch, sc, sh, rr, mr);
  for (int p = pb + threadIdx.y; p < pe; p += 4 * rows) {
    float v[4][V];
#pragma unroll
    for (int u = 0; u < 4; ++u)
      if (p + u * rows < pe) ldv(cat_ptr(p0, c0, p1, c1, (size_t)n * hw + p + u * rows, ch), v[u]);
#pragma unroll
    for (int u = 0; u < 4; ++u)
      if (p + u * rows < pe) {
#pragma unroll
        for (int i = 0; i < V; ++i) v[u][i] = siluf_(fmaf(v[u][i], sc[i], sh[i]));
        stv(out + ((size_t)n * hw + p + u * rows) * C + ch, v[u]);
      }
  }
}

// ------------------------------------------------------------------------------ backward: reduction pass
// bst[n][0][c] += sum_pix g_y, bst[n][1][c] += sum_pix g_y xhat
template <typename T>
__global__ void __launch_bounds__(512, 1)
gn_bwd_stats_k(const T* __restrict__ ga, const T* __restrict__ p0, int c0, const T* __restrict__ p1, int c1, int hw,
               int G, float eps, const T* __restrict__ gamma, const T* __restrict__ beta,
               const float* __restrict__ cst0, const float* __restrict__ cst1, float* __restrict__ bst) {
  constexpr int V = Vec<T>::N;
  extern __shared__ float sm_[];
  const int C = c0 + c1, n = blockIdx.y, nchunks = gridDim.x, rows = blockDim.y;
  Smem s(sm_, C, G);
  const int ppc = (hw + nchunks - 1) / nchunks;
  const int pb = blockIdx.x * ppc, pe = min(hw, pb + ppc);
  const int ch = threadIdx.x * V;
  group_mean_rstd(cst0, c0, cst1, c1, n, hw, G, eps, s);
  float sc[V], sh[V], rr[V], mr[V], v[2][V];
  gn_coefs<T, V>(s, G, C / G, gamma, beta, ch, sc, sh, rr, mr);
#pragma unroll
  for (int i = 0; i < V; ++i) v[0][i] = v[1][i] = 0.f;
  for (int p = pb + threadIdx.y; p < pe; p += 2 * rows) {
    float x[2][V], g[2][V];
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      if (p + u * rows < pe) {
        const size_t pix = (size_t)n * hw + p + u * rows;
        ldv(cat_ptr(p0, c0, p1, c1, pix, ch), x[u]);
        ldv(ga + pix * C + ch, g[u]);
      } else {
#pragma unroll
        for (int i = 0; i < V; ++i) { x[u][i] = 0.f; g[u][i] = 0.f; }
      }
    }
#pragma unroll
    for (int u = 0; u < 2; ++u)
#pragma unroll
      for (int i = 0; i < V; ++i) {
        const float gy = g[u][i] * silu_gradf_(fmaf(x[u][i], sc[i], sh[i]));
        v[0][i] += gy;
        v[1][i] = fmaf(gy, fmaf(x[u][i], rr[i], -mr[i]), v[1][i]);
      }
  }
  reduce_rows_atomic<V>(v, C, s, bst + (size_t)n * 2 * C);
}

// ------------------------------------------------------------------------------ backward: apply pass
// g_x = r (gamma g_y - A - xhat B) [+ add]; channels [0,dc0) -> dst0, the rest -> dst1 (skip gradient,
// PAPER.md:L91); acc: += instead of =.  cs0/cs1: per-(image, channel) sums of what this launch ADDS to
// dst0/dst1 (before bf16 rounding), accumulated.  dgamma/dbeta: += sum_n bst (CTA chunk 0 of each image).
template <typename T>
__global__ void __launch_bounds__(512, 1)
gn_bwd_apply_k(const T* __restrict__ ga, const T* __restrict__ p0, int c0, const T* __restrict__ p1, int c1, int hw,
               int G, float eps, const T* __restrict__ gamma, const T* __restrict__ beta,
               const float* __restrict__ cst0, const float* __restrict__ cst1, const float* __restrict__ bst,
               float* dgamma, float* dbeta, const T* __restrict__ add, T* dst0, int dc0, int acc0, T* dst1, int acc1,
               float* cs0, float* cs1) {
  constexpr int V = Vec<T>::N;
  extern __shared__ float sm_[];
  const int C = c0 + c1, n = blockIdx.y, nchunks = gridDim.x, rows = blockDim.y, cpg = C / G;
  Smem s(sm_, C, G);
  const int ppc = (hw + nchunks - 1) / nchunks;
  const int pb = blockIdx.x * ppc, pe = min(hw, pb + ppc);
  const int ch = threadIdx.x * V, tid = tid_(), nthr = nthr_();
  group_mean_rstd(cst0, c0, cst1, c1, n, hw, G, eps, s);
  float sc[V], sh[V], rr[V], mr[V], k2[V], k3[V];
  gn_coefs<T, V>(s, G, cpg, gamma, beta, ch, sc, sh, rr, mr);
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
  for (int p = pb + threadIdx.y; p < pe; p += 2 * rows) {
    float x[2][V], g[2][V], e[2][V], f[2][V];
#pragma unroll
    for (int u = 0; u < 2; ++u)
      if (p + u * rows < pe) {
        const size_t pix = (size_t)n * hw + p + u * rows;
        ldv(cat_ptr(p0, c0, p1, c1, pix, ch), x[u]);
        ldv(ga + pix * C + ch, g[u]);
        if (add) ldv(add + pix * C + ch, e[u]);
        if (acc) ldv(dst + pix * dC + dch, f[u]);
      }
#pragma unroll
    for (int u = 0; u < 2; ++u)
      if (p + u * rows < pe) {
        const size_t pix = (size_t)n * hw + p + u * rows;
        float o[V];
#pragma unroll
        for (int i = 0; i < V; ++i) {
          const float gy = g[u][i] * silu_gradf_(fmaf(x[u][i], sc[i], sh[i]));
          const float xh = fmaf(x[u][i], rr[i], -mr[i]);
          o[i] = sc[i] * gy - k2[i] - xh * k3[i];
          if (add) o[i] += e[u][i];
          sum[i] += o[i];
          if (acc) o[i] += f[u][i];
        }
        stv(dst + pix * dC + dch, o);
      }
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
int chan_stats(int dt, const void* x, int n, int hw, int c, float* cst, cudaStream_t st) {
  const RowPlan pl = row_plan(dt, hw, c, n, 512);
  dim3 grid(pl.nchunks, n), block(pl.tpr, pl.rows);
  const size_t sm = smem_bytes(c, 0, pl.rows, 2);
  if (dt == DT_F32) chan_stats_k<float><<<grid, block, sm, st>>>((const float*)x, c, hw, cst);
  else chan_stats_k<bf16><<<grid, block, sm, st>>>((const bf16*)x, c, hw, cst);
  return 1;
}

int gn_silu_fwd(int dt, Cat x, int n, int hw, int groups, float eps, const void* gamma, const void* beta,
                const float* cst0, const float* cst1, void* a_out, cudaStream_t st) {
  const int C = x.c();
  const RowPlan pl = row_plan(dt, hw, C, n, 512);
  dim3 grid(pl.nchunks, n), block(pl.tpr, pl.rows);
  const size_t sm = smem_bytes(C, groups, 1, 0);
  if (dt == DT_F32)
    gn_apply_k<float><<<grid, block, sm, st>>>((const float*)x.p0, x.c0, (const float*)x.p1, x.c1, hw, groups, eps,
                                               (const float*)gamma, (const float*)beta, cst0, cst1, (float*)a_out);
  else
    gn_apply_k<bf16><<<grid, block, sm, st>>>((const bf16*)x.p0, x.c0, (const bf16*)x.p1, x.c1, hw, groups, eps,
                                              (const bf16*)gamma, (const bf16*)beta, cst0, cst1, (bf16*)a_out);
  return 1;
}

template <typename T>
static int gn_bwd_t(const void* g_a, Cat x, int n, int hw, int groups, float eps, const void* gamma, const void* beta,
                    const float* cst0, const float* cst1, float* bst, const void* add, void* dst0, int dc0, int acc0,
                    void* dst1, int acc1, float* dgamma, float* dbeta, float* cs0, float* cs1, cudaStream_t st) {
  const int C = x.c();
  const int dt = sizeof(T) == 4 ? DT_F32 : DT_BF16;
  const RowPlan pl = row_plan(dt, hw, C, n, 256);
  dim3 grid(pl.nchunks, n), block(pl.tpr, pl.rows);
  static bool attr = false;
  if (!attr) {
    cudaFuncSetAttribute(gn_bwd_stats_k<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    cudaFuncSetAttribute(gn_bwd_apply_k<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    attr = true;
  }
  gn_bwd_stats_k<T><<<grid, block, smem_bytes(C, groups, pl.rows, 2), st>>>(
      (const T*)g_a, (const T*)x.p0, x.c0, (const T*)x.p1, x.c1, hw, groups, eps, (const T*)gamma, (const T*)beta, cst0,
      cst1, bst);
  gn_bwd_apply_k<T><<<grid, block, smem_bytes(C, groups, pl.rows, 1), st>>>(
      (const T*)g_a, (const T*)x.p0, x.c0, (const T*)x.p1, x.c1, hw, groups, eps, (const T*)gamma, (const T*)beta, cst0,
      cst1, bst, dgamma, dbeta, (const T*)add, (T*)dst0, dc0, acc0, (T*)dst1, acc1, cs0, cs1);
  return 2;
}

int gn_silu_bwd(int dt, const void* g_a, Cat x, int n, int hw, int groups, float eps, const void* gamma,
                const void* beta, const float* cst0, const float* cst1, float* bst, const void* add, void* dst0,
                int dc0, int acc0, void* dst1, int acc1, float* dgamma, float* dbeta, float* cs0, float* cs1,
                cudaStream_t st) {
  return dt == DT_F32 ? gn_bwd_t<float>(g_a, x, n, hw, groups, eps, gamma, beta, cst0, cst1, bst, add, dst0, dc0, acc0,
                                        dst1, acc1, dgamma, dbeta, cs0, cs1, st)
                      : gn_bwd_t<bf16>(g_a, x, n, hw, groups, eps, gamma, beta, cst0, cst1, bst, add, dst0, dc0, acc0,
                                       dst1, acc1, dgamma, dbeta, cs0, cs1, st);
}

}  // namespace pulse

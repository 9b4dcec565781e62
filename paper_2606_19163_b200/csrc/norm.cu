// norm.cu - fused GroupNorm + SiLU forward / backward on NHWC tensors, single or
// dual source (virtual concat).  SURVEY.md 8c item 1:
//   fwd: mu, var per (n,group) (biased), r = rsqrt(var+eps), xhat = (x-mu) r,
//        y = gamma xhat + beta, a = y sigmoid(y)
//   bwd: g_y = g_a SiLU'(y); dgamma = sum g_y xhat; dbeta = sum g_y; q = g_y gamma;
//        A = mean_S q; B = mean_S q xhat; g_x = r (q - A - xhat B)
// Layout choice for NHWC: a thread owns one 16-byte channel vector and walks pixels, so
// every warp-wide access is contiguous and per-channel partial sums live in registers;
// group statistics are then formed from per-channel sums in a tiny finalize kernel
// (groups of 10/20/30/60 channels are not 16-byte aligned and may straddle the h|skip
// boundary - per-channel partials make both irrelevant).
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

GnPlan gn_plan(int dt, int hw, int c, int n) {
  GnPlan p;
  const int vec = dt == DT_F32 ? 4 : 8;
  p.tpr = c / vec;
  p.rows = p.tpr >= 256 ? 1 : 256 / p.tpr;
  if (p.rows > hw) p.rows = hw;
  // ~2 CTAs per SM, at least 8 pixels per thread row (4 loads in flight x 2)
  int want = (2 * num_sms() + n - 1) / n;
  int maxc = hw / (p.rows * 8);
  if (maxc < 1) maxc = 1;
  p.nchunks = want < maxc ? want : maxc;
  return p;
}
// scratch floats: per-CTA group partials [n][chunk][G][2] + per-CTA channel partials [n][chunk][2][C]
size_t gn_partial_elems(const GnPlan& p, int n, int c) { return (size_t)n * p.nchunks * (2 * (size_t)c + 2 * 64) + 1024; }

template <typename T>
__device__ __forceinline__ const T* cat_ptr(const T* p0, int c0, const T* p1, int c1, size_t pix, int ch) {
  return ch < c0 ? p0 + pix * c0 + ch : p1 + pix * c1 + (ch - c0);
}

// Cross-CTA reductions avoid same-address atomics (hundreds of CTAs adding into C addresses serialise
// in L2, measured 30 us for a 10 MB tensor): every CTA writes its partials, and the consuming kernel
// finalises them in its prologue - group sums redundantly per CTA (2G values x nchunks loads), channel
// sums with each channel owned by exactly one CTA.

// sm_g[2G] doubles <- sum over chunks of pg[n][chunk][2G]
__device__ __forceinline__ void group_sums_to_smem(const float* __restrict__ pg, int n, int nchunks, int G, double* sm_g) {
  const int tid = threadIdx.y * blockDim.x + threadIdx.x, nthr = blockDim.x * blockDim.y;
  for (int i = tid; i < 2 * G; i += nthr) {
    const float* p = pg + (size_t)n * nchunks * 2 * G + i;
    double s = 0.0;
    for (int k = 0; k < nchunks; ++k) s += (double)p[(size_t)k * 2 * G];
    sm_g[i] = s;
  }
  __syncthreads();
}

// per-thread normalisation coefficients of V consecutive channels from the group sums (sum, sum of squares)
template <typename T, int V>
__device__ __forceinline__ void gn_coefs(const double* gsum_n, int cpg, int hw, float eps, const T* __restrict__ gamma,
                                         const T* __restrict__ beta, int ch, float (&sc)[V], float (&sh)[V],
                                         float (&rr)[V], float (&mr)[V]) {
  const double m = (double)cpg * hw;
#pragma unroll
  for (int i = 0; i < V; ++i) {
    const int g = (ch + i) / cpg;
    const double mu = gsum_n[2 * g] / m;
    double var = gsum_n[2 * g + 1] / m - mu * mu;
    if (var < 0.0) var = 0.0;
    const float r = (float)(1.0 / sqrt(var + (double)eps));
    const float ga = to_f(gamma[ch + i]), be = to_f(beta[ch + i]);
    rr[i] = r; mr[i] = (float)mu * r;
    sc[i] = r * ga; sh[i] = be - mr[i] * ga;
  }
}

// block-reduce per-channel partials over rows; write per-group partials pg_out[2G] (weighted by wgt) and,
// if pc_out, the per-channel sums pc_out[0..C) = s1, pc_out[C..2C) = s2
template <int V, typename T>
__device__ __forceinline__ void reduce_block(float (&s1)[V], float (&s2)[V], int C, int G, int cpg, const T* wgt,
                                             float* pg_out, float* pc_out) {
  extern __shared__ float sm[];
  const int rows = blockDim.y, tx = threadIdx.x, ty = threadIdx.y, ch = tx * V;
  float* a = sm;                  // [rows][C]
  float* b = sm + rows * C;       // [rows][C]
  float* gs = sm + 2 * rows * C;  // [G][2]
  const int tid = ty * blockDim.x + tx, nthr = blockDim.x * blockDim.y;
  for (int i = tid; i < 2 * G; i += nthr) gs[i] = 0.f;
  if (rows > 1) {
#pragma unroll
    for (int i = 0; i < V; ++i) { a[ty * C + ch + i] = s1[i]; b[ty * C + ch + i] = s2[i]; }
  }
  __syncthreads();
  if (ty == 0) {
#pragma unroll
    for (int i = 0; i < V; ++i) {
      float u = s1[i], v = s2[i];
      if (rows > 1) {
        u = 0.f; v = 0.f;
        for (int r = 0; r < rows; ++r) { u += a[r * C + ch + i]; v += b[r * C + ch + i]; }
      }
      if (pc_out) { pc_out[ch + i] = u; pc_out[C + ch + i] = v; }
      const float w = wgt ? to_f(wgt[ch + i]) : 1.f;
      const int g = (ch + i) / cpg;
      atomicAdd(&gs[2 * g], w * u);        // shared-memory atomics, <= cpg-way
      atomicAdd(&gs[2 * g + 1], w * v);
    }
  }
  __syncthreads();
  for (int i = tid; i < 2 * G; i += nthr) pg_out[i] = gs[i];
}

template <typename T>
__global__ void __launch_bounds__(512) gn_stats_k(const T* __restrict__ p0, int c0, const T* __restrict__ p1, int c1,
                                                  int hw, int G, float* __restrict__ pg) {
  constexpr int V = Vec<T>::N;
  const int C = c0 + c1, n = blockIdx.y, chunk = blockIdx.x, nchunks = gridDim.x;
  const int ppc = (hw + nchunks - 1) / nchunks;
  const int pb = chunk * ppc, pe = min(hw, pb + ppc);
  const int ch = threadIdx.x * V, rows = blockDim.y;
  float s1[V], s2[V];
#pragma unroll
  for (int i = 0; i < V; ++i) s1[i] = s2[i] = 0.f;
  for (int p = pb + threadIdx.y; p < pe; p += 4 * rows) {
    float v[4][V];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      if (p + u * rows < pe) ldv(cat_ptr(p0, c0, p1, c1, (size_t)n * hw + p + u * rows, ch), v[u]);
      else {
#pragma unroll
        for (int i = 0; i < V; ++i) v[u][i] = 0.f;
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int i = 0; i < V; ++i) { s1[i] += v[u][i]; s2[i] = fmaf(v[u][i], v[u][i], s2[i]); }
  }
  reduce_block<V, T>(s1, s2, C, G, C / G, nullptr, pg + ((size_t)n * nchunks + chunk) * 2 * G, nullptr);
}

template <typename T>
__global__ void __launch_bounds__(512) gn_silu_apply_k(const T* __restrict__ p0, int c0, const T* __restrict__ p1, int c1,
                                                       int hw, int G, float eps, const T* __restrict__ gamma,
                                                       const T* __restrict__ beta, const float* __restrict__ pg,
                                                       double* __restrict__ gsum, T* __restrict__ out) {
  constexpr int V = Vec<T>::N;
  __shared__ double sm_g[128];
  const int C = c0 + c1, n = blockIdx.y, chunk = blockIdx.x, nchunks = gridDim.x;
  const int ppc = (hw + nchunks - 1) / nchunks;
  const int pb = chunk * ppc, pe = min(hw, pb + ppc);
  const int ch = threadIdx.x * V, rows = blockDim.y;
  group_sums_to_smem(pg, n, nchunks, G, sm_g);
  if (chunk == 0) {     // keep the group sums for the backward pass
    const int tid = threadIdx.y * blockDim.x + threadIdx.x;
    for (int i = tid; i < 2 * G; i += blockDim.x * blockDim.y) gsum[(size_t)n * 2 * G + i] = sm_g[i];
  }
  float sc[V], sh[V], rr[V], mr[V];
  gn_coefs<T, V>(sm_g, C / G, hw, eps, gamma, beta, ch, sc, sh, rr, mr);
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

static size_t gn_smem(const GnPlan& pl, int C, int G) { return ((size_t)2 * pl.rows * C + 2 * G) * sizeof(float); }

template <typename T>
static int gn_fwd_t(Cat x, int n, int hw, int groups, float eps, const void* gamma, const void* beta, void* a_out,
                    double* gsum, float* partial, const GnPlan& pl, cudaStream_t st) {
  const int C = x.c();
  dim3 grid(pl.nchunks, n), block(pl.tpr, pl.rows);
  gn_stats_k<T><<<grid, block, gn_smem(pl, C, groups), st>>>((const T*)x.p0, x.c0, (const T*)x.p1, x.c1, hw, groups, partial);
  gn_silu_apply_k<T><<<grid, block, 0, st>>>((const T*)x.p0, x.c0, (const T*)x.p1, x.c1, hw, groups, eps,
                                             (const T*)gamma, (const T*)beta, partial, gsum, (T*)a_out);
  return 2;
}

int gn_silu_fwd(int dt, Cat x, int n, int hw, int groups, float eps, const void* gamma, const void* beta,
                void* a_out, double* gsum, float* partial, cudaStream_t st) {
  GnPlan pl = gn_plan(dt, hw, x.c(), n);
  return dt == DT_F32 ? gn_fwd_t<float>(x, n, hw, groups, eps, gamma, beta, a_out, gsum, partial, pl, st)
                      : gn_fwd_t<bf16>(x, n, hw, groups, eps, gamma, beta, a_out, gsum, partial, pl, st);
}

// ------------------------------------------------------------------------------ backward

template <typename T>
__global__ void __launch_bounds__(512) gn_bwd_stats_k(const T* __restrict__ ga, const T* __restrict__ p0, int c0,
                                                      const T* __restrict__ p1, int c1, int hw, int G, float eps,
                                                      const T* __restrict__ gamma, const T* __restrict__ beta,
                                                      const double* __restrict__ gsum, float* __restrict__ pg,
                                                      float* __restrict__ pc) {
  constexpr int V = Vec<T>::N;
  const int C = c0 + c1, n = blockIdx.y, chunk = blockIdx.x, nchunks = gridDim.x;
  const int ppc = (hw + nchunks - 1) / nchunks;
  const int pb = chunk * ppc, pe = min(hw, pb + ppc);
  const int ch = threadIdx.x * V, rows = blockDim.y;
  float sc[V], sh[V], rr[V], mr[V], s1[V], s2[V];
  gn_coefs<T, V>(gsum + (size_t)n * 2 * G, C / G, hw, eps, gamma, beta, ch, sc, sh, rr, mr);
#pragma unroll
  for (int i = 0; i < V; ++i) s1[i] = s2[i] = 0.f;
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
        s1[i] += gy;
        s2[i] = fmaf(gy, fmaf(x[u][i], rr[i], -mr[i]), s2[i]);
      }
  }
  // channel partials: s1 -> dbeta, s2 -> dgamma; group partials weighted by gamma: A m = sum gamma s1, B m = sum gamma s2
  const size_t cta = (size_t)n * nchunks + chunk;
  reduce_block<V, T>(s1, s2, C, G, C / G, gamma, pg + cta * 2 * G, pc + cta * 2 * C);
}

template <typename T>
__global__ void __launch_bounds__(512) gn_bwd_apply_k(const T* __restrict__ ga, const T* __restrict__ p0, int c0,
                                                      const T* __restrict__ p1, int c1, int hw, int G, float eps,
                                                      const T* __restrict__ gamma, const T* __restrict__ beta,
                                                      const double* __restrict__ gsum, const float* __restrict__ pg,
                                                      const float* __restrict__ pc, float* dgamma, float* dbeta,
                                                      const T* __restrict__ add, T* dst0, int dc0, int acc0, T* dst1,
                                                      int acc1) {
  constexpr int V = Vec<T>::N;
  __shared__ double sm_g[128];
  const int C = c0 + c1, n = blockIdx.y, chunk = blockIdx.x, nchunks = gridDim.x, cpg = C / G;
  const int ppc = (hw + nchunks - 1) / nchunks;
  const int pb = chunk * ppc, pe = min(hw, pb + ppc);
  const int ch = threadIdx.x * V, rows = blockDim.y;
  group_sums_to_smem(pg, n, nchunks, G, sm_g);
  {  // dgamma / dbeta: (channel, which) pair j is owned by CTA j % T; one warp sums its T partial rows
    const int T_ = gridDim.x * gridDim.y, cta = blockIdx.y * gridDim.x + blockIdx.x;
    const int tid = threadIdx.y * blockDim.x + threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthr = blockDim.x * blockDim.y, nwarps = (nthr + 31) >> 5;
    const bool full = (warp + 1) * 32 <= nthr;      // a partial last warp sums serially on its lane 0
    for (int j = cta + warp * T_; j < 2 * C; j += nwarps * T_) {
      const int which = j / C, c = j - which * C;
      float s = 0.f;
      if (full) {
        for (int r = lane; r < T_; r += 32) s += pc[(size_t)r * 2 * C + which * C + c];
        s = warp_sum(s);
      } else if (lane == 0) {
        for (int r = 0; r < T_; ++r) s += pc[(size_t)r * 2 * C + which * C + c];
      }
      if (lane == 0) {
        if (which) dgamma[c] += s; else dbeta[c] += s;
      }
    }
  }
  float sc[V], sh[V], rr[V], mr[V], k2[V], k3[V];
  gn_coefs<T, V>(gsum + (size_t)n * 2 * G, cpg, hw, eps, gamma, beta, ch, sc, sh, rr, mr);
  const double m = (double)cpg * hw;
#pragma unroll
  for (int i = 0; i < V; ++i) {
    const int g = (ch + i) / cpg;
    k2[i] = (float)(sm_g[2 * g] / m) * rr[i];
    k3[i] = (float)(sm_g[2 * g + 1] / m) * rr[i];
  }
  const bool first = ch < dc0;
  T* dst = first ? dst0 : dst1;
  const int dC = first ? dc0 : C - dc0, dch = first ? ch : ch - dc0;
  const int acc = first ? acc0 : acc1;
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
          if (acc) o[i] += f[u][i];
        }
        stv(dst + pix * dC + dch, o);
      }
  }
}

template <typename T>
static int gn_bwd_t(const void* g_a, Cat x, int n, int hw, int groups, float eps, const void* gamma, const void* beta,
                    const double* gsum, const void* add, void* dst0, int dc0, int acc0, void* dst1, int acc1,
                    float* dgamma, float* dbeta, float* partial, const GnPlan& pl, cudaStream_t st) {
  const int C = x.c();
  dim3 grid(pl.nchunks, n), block(pl.tpr, pl.rows);
  float* pg = partial;
  float* pc = partial + (size_t)n * pl.nchunks * 2 * groups;
  gn_bwd_stats_k<T><<<grid, block, gn_smem(pl, C, groups), st>>>((const T*)g_a, (const T*)x.p0, x.c0, (const T*)x.p1, x.c1,
                                                                  hw, groups, eps, (const T*)gamma, (const T*)beta, gsum, pg, pc);
  gn_bwd_apply_k<T><<<grid, block, 0, st>>>((const T*)g_a, (const T*)x.p0, x.c0, (const T*)x.p1, x.c1, hw, groups, eps,
                                            (const T*)gamma, (const T*)beta, gsum, pg, pc, dgamma, dbeta, (const T*)add,
                                            (T*)dst0, dc0, acc0, (T*)dst1, acc1);
  return 2;
}

int gn_silu_bwd(int dt, const void* g_a, Cat x, int n, int hw, int groups, float eps, const void* gamma,
                const void* beta, const double* gsum, const void* add, void* dst0, int dc0, int acc0, void* dst1,
                int acc1, float* dgamma, float* dbeta, float* partial, cudaStream_t st) {
  GnPlan pl = gn_plan(dt, hw, x.c(), n);
  return dt == DT_F32 ? gn_bwd_t<float>(g_a, x, n, hw, groups, eps, gamma, beta, gsum, add, dst0, dc0, acc0, dst1, acc1,
                                        dgamma, dbeta, partial, pl, st)
                      : gn_bwd_t<bf16>(g_a, x, n, hw, groups, eps, gamma, beta, gsum, add, dst0, dc0, acc0, dst1, acc1,
                                       dgamma, dbeta, partial, pl, st);
}

}  // namespace pulse

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
  // enough CTAs for ~4 per SM, but at least 4 pixels per thread row
  int want = (4 * num_sms() + n - 1) / n;
  int maxc = hw / (p.rows * 4);
  if (maxc < 1) maxc = 1;
  p.nchunks = want < maxc ? want : maxc;
  return p;
}
size_t gn_partial_elems(const GnPlan& p, int n, int c) { return (size_t)n * p.nchunks * 2 * c; }

template <typename T>
__device__ __forceinline__ const T* cat_ptr(const T* p0, int c0, const T* p1, int c1, size_t pix, int ch) {
  return ch < c0 ? p0 + pix * c0 + ch : p1 + pix * c1 + (ch - c0);
}

// reduce per-thread per-channel partials over the `rows` dimension and store
template <int V>
__device__ __forceinline__ void reduce_rows_store(float (&s1)[V], float (&s2)[V], float* out1, float* out2, int C) {
  extern __shared__ float sm[];
  const int tpr = blockDim.x, rows = blockDim.y, tx = threadIdx.x, ty = threadIdx.y;
  if (rows > 1) {
    float* a = sm;
    float* b = sm + rows * C;
#pragma unroll
    for (int i = 0; i < V; ++i) {
      a[ty * C + tx * V + i] = s1[i];
      b[ty * C + tx * V + i] = s2[i];
    }
    __syncthreads();
    if (ty == 0) {
#pragma unroll
      for (int i = 0; i < V; ++i) {
        float u = 0.f, v = 0.f;
        for (int r = 0; r < rows; ++r) {
          u += a[r * C + tx * V + i];
          v += b[r * C + tx * V + i];
        }
        s1[i] = u; s2[i] = v;
      }
    }
  }
  if (ty == 0) {
#pragma unroll
    for (int i = 0; i < V; ++i) {
      out1[tx * V + i] = s1[i];
      out2[tx * V + i] = s2[i];
    }
  }
  (void)tpr;
}

template <typename T>
__global__ void gn_stats_partial_k(const T* __restrict__ p0, int c0, const T* __restrict__ p1, int c1, int hw,
                                   float* __restrict__ partial) {
  constexpr int V = Vec<T>::N;
  const int C = c0 + c1, n = blockIdx.y, chunk = blockIdx.x, nchunks = gridDim.x;
  const int ppc = (hw + nchunks - 1) / nchunks;
  const int pb = chunk * ppc, pe = min(hw, pb + ppc);
  const int ch = threadIdx.x * V;
  float s1[V], s2[V];
#pragma unroll
  for (int i = 0; i < V; ++i) s1[i] = s2[i] = 0.f;
  for (int p = pb + threadIdx.y; p < pe; p += blockDim.y) {
    float v[V];
    ldv(cat_ptr(p0, c0, p1, c1, (size_t)n * hw + p, ch), v);
#pragma unroll
    for (int i = 0; i < V; ++i) { s1[i] += v[i]; s2[i] += v[i] * v[i]; }
  }
  float* o = partial + ((size_t)n * nchunks + chunk) * 2 * C;
  reduce_rows_store<V>(s1, s2, o, o + C, C);
}

template <typename T>
__global__ void gn_stats_finalize_k(const float* __restrict__ partial, int nchunks, int C, int groups, int hw,
                                    float eps, const T* __restrict__ gamma, const T* __restrict__ beta,
                                    float* __restrict__ stats) {
  const int g = blockIdx.x, n = blockIdx.y, cpg = C / groups;
  double s1 = 0.0, s2 = 0.0;
  for (int i = threadIdx.x; i < nchunks * cpg; i += blockDim.x) {
    const int chunk = i / cpg, c = g * cpg + i % cpg;
    const float* o = partial + ((size_t)n * nchunks + chunk) * 2 * C;
    s1 += (double)o[c];
    s2 += (double)o[C + c];
  }
  __shared__ double sh1[32], sh2[32];
  for (int o = 16; o > 0; o >>= 1) {
    s1 += __shfl_xor_sync(0xffffffffu, s1, o);
    s2 += __shfl_xor_sync(0xffffffffu, s2, o);
  }
  const int wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  if ((threadIdx.x & 31) == 0) { sh1[wid] = s1; sh2[wid] = s2; }
  __syncthreads();
  s1 = 0.0; s2 = 0.0;
  for (int i = 0; i < nw; ++i) { s1 += sh1[i]; s2 += sh2[i]; }
  const double m = (double)cpg * hw;
  const double mu = s1 / m;
  double var = s2 / m - mu * mu;
  if (var < 0.0) var = 0.0;
  const float r = (float)(1.0 / sqrt(var + (double)eps));
  const float mur = (float)mu * r;
  float* sn = stats + (size_t)n * 4 * C;
  for (int i = threadIdx.x; i < cpg; i += blockDim.x) {
    const int c = g * cpg + i;
    const float ga = to_f(gamma[c]), be = to_f(beta[c]);
    sn[c] = r * ga;
    sn[C + c] = be - mur * ga;
    sn[2 * C + c] = r;
    sn[3 * C + c] = mur;
  }
}

template <typename T>
__global__ void gn_silu_apply_k(const T* __restrict__ p0, int c0, const T* __restrict__ p1, int c1, int hw,
                                const float* __restrict__ stats, T* __restrict__ out) {
  constexpr int V = Vec<T>::N;
  const int C = c0 + c1, n = blockIdx.y, chunk = blockIdx.x, nchunks = gridDim.x;
  const int ppc = (hw + nchunks - 1) / nchunks;
  const int pb = chunk * ppc, pe = min(hw, pb + ppc);
  const int ch = threadIdx.x * V;
  float sc[V], sh[V];
  const float* sn = stats + (size_t)n * 4 * C;
#pragma unroll
  for (int i = 0; i < V; ++i) { sc[i] = sn[ch + i]; sh[i] = sn[C + ch + i]; }
  for (int p = pb + threadIdx.y; p < pe; p += blockDim.y) {
    const size_t pix = (size_t)n * hw + p;
    float v[V];
    ldv(cat_ptr(p0, c0, p1, c1, pix, ch), v);
#pragma unroll
    for (int i = 0; i < V; ++i) v[i] = siluf_(fmaf(v[i], sc[i], sh[i]));
    stv(out + pix * C + ch, v);
  }
}

template <typename T>
static int gn_fwd_t(Cat x, int n, int hw, int groups, float eps, const void* gamma, const void* beta, void* a_out,
                    float* stats, float* partial, const GnPlan& pl, cudaStream_t st) {
  const int C = x.c();
  dim3 grid(pl.nchunks, n), block(pl.tpr, pl.rows);
  const size_t smem = pl.rows > 1 ? (size_t)pl.rows * C * 2 * sizeof(float) : 0;
  gn_stats_partial_k<T><<<grid, block, smem, st>>>((const T*)x.p0, x.c0, (const T*)x.p1, x.c1, hw, partial);
  gn_stats_finalize_k<T><<<dim3(groups, n), 128, 0, st>>>(partial, pl.nchunks, C, groups, hw, eps, (const T*)gamma,
                                                           (const T*)beta, stats);
  gn_silu_apply_k<T><<<grid, block, 0, st>>>((const T*)x.p0, x.c0, (const T*)x.p1, x.c1, hw, stats, (T*)a_out);
  return 3;
}

int gn_silu_fwd(int dt, Cat x, int n, int hw, int groups, float eps, const void* gamma, const void* beta,
                void* a_out, float* stats, float* partial, cudaStream_t st) {
  GnPlan pl = gn_plan(dt, hw, x.c(), n);
  return dt == DT_F32 ? gn_fwd_t<float>(x, n, hw, groups, eps, gamma, beta, a_out, stats, partial, pl, st)
                      : gn_fwd_t<bf16>(x, n, hw, groups, eps, gamma, beta, a_out, stats, partial, pl, st);
}

// ------------------------------------------------------------------------------ backward

template <typename T>
__global__ void gn_bwd_partial_k(const T* __restrict__ ga, const T* __restrict__ p0, int c0,
                                 const T* __restrict__ p1, int c1, int hw, const float* __restrict__ stats,
                                 float* __restrict__ partial) {
  constexpr int V = Vec<T>::N;
  const int C = c0 + c1, n = blockIdx.y, chunk = blockIdx.x, nchunks = gridDim.x;
  const int ppc = (hw + nchunks - 1) / nchunks;
  const int pb = chunk * ppc, pe = min(hw, pb + ppc);
  const int ch = threadIdx.x * V;
  const float* sn = stats + (size_t)n * 4 * C;
  float sc[V], sh[V], rr[V], mr[V], s1[V], s2[V];
#pragma unroll
  for (int i = 0; i < V; ++i) {
    sc[i] = sn[ch + i]; sh[i] = sn[C + ch + i]; rr[i] = sn[2 * C + ch + i]; mr[i] = sn[3 * C + ch + i];
    s1[i] = s2[i] = 0.f;
  }
  for (int p = pb + threadIdx.y; p < pe; p += blockDim.y) {
    const size_t pix = (size_t)n * hw + p;
    float x[V], g[V];
    ldv(cat_ptr(p0, c0, p1, c1, pix, ch), x);
    ldv(ga + pix * C + ch, g);
#pragma unroll
    for (int i = 0; i < V; ++i) {
      const float gy = g[i] * silu_gradf_(fmaf(x[i], sc[i], sh[i]));
      s1[i] += gy;
      s2[i] += gy * fmaf(x[i], rr[i], -mr[i]);
    }
  }
  float* o = partial + ((size_t)n * nchunks + chunk) * 2 * C;
  reduce_rows_store<V>(s1, s2, o, o + C, C);
}

template <typename T>
__global__ void gn_bwd_finalize_k(const float* __restrict__ partial, int nchunks, int C, int groups, int hw,
                                  const T* __restrict__ gamma, const float* __restrict__ stats,
                                  float* __restrict__ dgamma, float* __restrict__ dbeta, float* __restrict__ coef) {
  const int g = blockIdx.x, n = blockIdx.y, cpg = C / groups;
  extern __shared__ float sm[];      // [2][cpg] per-channel sums
  for (int i = threadIdx.x; i < cpg; i += blockDim.x) {
    const int c = g * cpg + i;
    float a = 0.f, b = 0.f;
    for (int k = 0; k < nchunks; ++k) {
      const float* o = partial + ((size_t)n * nchunks + k) * 2 * C;
      a += o[c];
      b += o[C + c];
    }
    sm[i] = a; sm[cpg + i] = b;
    atomicAdd(dbeta + c, a);
    atomicAdd(dgamma + c, b);
  }
  __syncthreads();
  double A = 0.0, B = 0.0;
  for (int i = 0; i < cpg; ++i) {          // cpg <= 80: serial per thread, no second reduction
    const float gm = to_f(gamma[g * cpg + i]);
    A += (double)gm * sm[i];
    B += (double)gm * sm[cpg + i];
  }
  const double m = (double)cpg * hw;
  const float r = stats[(size_t)n * 4 * C + 2 * C + g * cpg];
  const float c2 = (float)(A / m) * r, c3 = (float)(B / m) * r;
  float* cn = coef + (size_t)n * 2 * C;
  for (int i = threadIdx.x; i < cpg; i += blockDim.x) {
    cn[g * cpg + i] = c2;
    cn[C + g * cpg + i] = c3;
  }
}

template <typename T>
__global__ void gn_bwd_apply_k(const T* __restrict__ ga, const T* __restrict__ p0, int c0,
                               const T* __restrict__ p1, int c1, int hw, const float* __restrict__ stats,
                               const float* __restrict__ coef, const T* __restrict__ add, T* dst0, int dc0, int acc0,
                               T* dst1, int acc1) {
  constexpr int V = Vec<T>::N;
  const int C = c0 + c1, n = blockIdx.y, chunk = blockIdx.x, nchunks = gridDim.x;
  const int ppc = (hw + nchunks - 1) / nchunks;
  const int pb = chunk * ppc, pe = min(hw, pb + ppc);
  const int ch = threadIdx.x * V;
  const float* sn = stats + (size_t)n * 4 * C;
  const float* cn = coef + (size_t)n * 2 * C;
  float sc[V], sh[V], rr[V], mr[V], k2[V], k3[V];
#pragma unroll
  for (int i = 0; i < V; ++i) {
    sc[i] = sn[ch + i]; sh[i] = sn[C + ch + i]; rr[i] = sn[2 * C + ch + i]; mr[i] = sn[3 * C + ch + i];
    k2[i] = cn[ch + i]; k3[i] = cn[C + ch + i];
  }
  const bool first = ch < dc0;
  T* dst = first ? dst0 : dst1;
  const int dC = first ? dc0 : C - dc0, dch = first ? ch : ch - dc0;
  const int acc = first ? acc0 : acc1;
  for (int p = pb + threadIdx.y; p < pe; p += blockDim.y) {
    const size_t pix = (size_t)n * hw + p;
    float x[V], g[V], o[V];
    ldv(cat_ptr(p0, c0, p1, c1, pix, ch), x);
    ldv(ga + pix * C + ch, g);
#pragma unroll
    for (int i = 0; i < V; ++i) {
      const float gy = g[i] * silu_gradf_(fmaf(x[i], sc[i], sh[i]));
      const float xh = fmaf(x[i], rr[i], -mr[i]);
      o[i] = sc[i] * gy - k2[i] - xh * k3[i];
    }
    if (add) {
      float e[V];
      ldv(add + pix * C + ch, e);
#pragma unroll
      for (int i = 0; i < V; ++i) o[i] += e[i];
    }
    T* d = dst + pix * dC + dch;
    if (acc) {
      float e[V];
      ldv(d, e);
#pragma unroll
      for (int i = 0; i < V; ++i) o[i] += e[i];
    }
    stv(d, o);
  }
}

template <typename T>
static int gn_bwd_t(const void* g_a, Cat x, int n, int hw, int groups, const void* gamma, const float* stats,
                    const void* add, void* dst0, int dc0, int acc0, void* dst1, int acc1, float* dgamma,
                    float* dbeta, float* partial, float* coef, const GnPlan& pl, cudaStream_t st) {
  const int C = x.c();
  dim3 grid(pl.nchunks, n), block(pl.tpr, pl.rows);
  const size_t smem = pl.rows > 1 ? (size_t)pl.rows * C * 2 * sizeof(float) : 0;
  gn_bwd_partial_k<T><<<grid, block, smem, st>>>((const T*)g_a, (const T*)x.p0, x.c0, (const T*)x.p1, x.c1, hw,
                                                  stats, partial);
  const int cpg = C / groups;
  gn_bwd_finalize_k<T><<<dim3(groups, n), 64, 2 * cpg * sizeof(float), st>>>(partial, pl.nchunks, C, groups, hw,
                                                                             (const T*)gamma, stats, dgamma, dbeta,
                                                                             coef);
  gn_bwd_apply_k<T><<<grid, block, 0, st>>>((const T*)g_a, (const T*)x.p0, x.c0, (const T*)x.p1, x.c1, hw, stats,
                                            coef, (const T*)add, (T*)dst0, dc0, acc0, (T*)dst1, acc1);
  return 3;
}

int gn_silu_bwd(int dt, const void* g_a, Cat x, int n, int hw, int groups, const void* gamma, const float* stats,
                const void* add, void* dst0, int dc0, int acc0, void* dst1, int acc1, float* dgamma, float* dbeta,
                float* partial, float* coef, cudaStream_t st) {
  GnPlan pl = gn_plan(dt, hw, x.c(), n);
  return dt == DT_F32 ? gn_bwd_t<float>(g_a, x, n, hw, groups, gamma, stats, add, dst0, dc0, acc0, dst1, acc1,
                                        dgamma, dbeta, partial, coef, pl, st)
                      : gn_bwd_t<bf16>(g_a, x, n, hw, groups, gamma, stats, add, dst0, dc0, acc0, dst1, acc1,
                                       dgamma, dbeta, partial, coef, pl, st);
}

}  // namespace pulse

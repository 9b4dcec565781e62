// tblock.cu - the pointwise kernels of the transformer block with a long skip (
// formulas: oracle ln_fwd / ln_bwd / gelu / gelu_grad).  The block's Linear layers are 1x1 convs on the tcgen05 conv
// path (the long skip "concat + Linear" is the 1x1 conv on the virtual concat), its attention is attention(_tc).cu.
//   LayerNorm over the C channels of every token (pixel of an NHWC tensor): one warp per token, the row is read three
//   times from L1 (mean, centred variance, apply) - C <= 1280 channels = 2.5 KB per row; mean / rstd are saved per token.
//   Backward: g_x = r (q - mean_c q - xhat mean_c (q xhat)) [+ add], q = g_y gamma; dgamma / dbeta are summed per CTA in
//   shared memory and added to the fp32 gradients with one atomic per channel and CTA.
//   GELU: the exact erf form, elementwise.
#include "common.cuh"
#include "kernels.h"

namespace pulse {

namespace {

constexpr int LN_WARPS = 8;

template <typename T>
__global__ void __launch_bounds__(LN_WARPS * 32) ln_fwd_k(const T* __restrict__ x, int C, size_t tokens, float eps,
                                                           const T* __restrict__ gamma, const T* __restrict__ beta,
                                                           float* __restrict__ stat, T* __restrict__ y) {
  constexpr int V = Vec<T>::N;
  const int lane = threadIdx.x & 31, nvec = C / V;
  for (size_t t = (size_t)blockIdx.x * LN_WARPS + (threadIdx.x >> 5); t < tokens; t += (size_t)gridDim.x * LN_WARPS) {
    const T* row = x + t * C;
    float s = 0.f;
    for (int v = lane; v < nvec; v += 32) {
      float a[V];
      ldv(row + v * V, a);
#pragma unroll
      for (int i = 0; i < V; ++i) s += a[i];
    }
    const float mu = warp_sum(s) / (float)C;
    float q = 0.f;
    for (int v = lane; v < nvec; v += 32) {
      float a[V];
      ldv(row + v * V, a);
#pragma unroll
      for (int i = 0; i < V; ++i) q = fmaf(a[i] - mu, a[i] - mu, q);
    }
    const float r = rsqrtf(warp_sum(q) / (float)C + eps);
    if (lane == 0) { stat[2 * t] = mu; stat[2 * t + 1] = r; }
    for (int v = lane; v < nvec; v += 32) {
      float a[V], g[V], b[V];
      ldv(row + v * V, a); ldv(gamma + v * V, g); ldv(beta + v * V, b);
#pragma unroll
      for (int i = 0; i < V; ++i) a[i] = fmaf((a[i] - mu) * r, g[i], b[i]);
      stv(y + t * C + v * V, a);
    }
  }
}

template <typename T>
__global__ void __launch_bounds__(LN_WARPS * 32) ln_bwd_k(const T* __restrict__ gy, const T* __restrict__ x, int C, size_t tokens,
                                                           const T* __restrict__ gamma, const float* __restrict__ stat,
                                                           const T* __restrict__ add, T* __restrict__ gx, int acc,
                                                           float* __restrict__ dgamma, float* __restrict__ dbeta) {
  constexpr int V = Vec<T>::N;
  extern __shared__ float sm[];            // [2][C]: dgamma | dbeta of this CTA
  for (int i = threadIdx.x; i < 2 * C; i += blockDim.x) sm[i] = 0.f;
  __syncthreads();
  const int lane = threadIdx.x & 31, nvec = C / V;
  for (size_t t = (size_t)blockIdx.x * LN_WARPS + (threadIdx.x >> 5); t < tokens; t += (size_t)gridDim.x * LN_WARPS) {
    const float mu = stat[2 * t], r = stat[2 * t + 1];
    float s1 = 0.f, s2 = 0.f;
    for (int v = lane; v < nvec; v += 32) {
      float a[V], g[V], ga[V];
      ldv(x + t * C + v * V, a); ldv(gy + t * C + v * V, g); ldv(gamma + v * V, ga);
#pragma unroll
      for (int i = 0; i < V; ++i) {
        const float xh = (a[i] - mu) * r, q = g[i] * ga[i];
        s1 += q; s2 = fmaf(q, xh, s2);
        atomicAdd(&sm[v * V + i], g[i] * xh);
        atomicAdd(&sm[C + v * V + i], g[i]);
      }
    }
    const float m1 = warp_sum(s1) / (float)C, m2 = warp_sum(s2) / (float)C;
    for (int v = lane; v < nvec; v += 32) {
      float a[V], g[V], ga[V], o[V];
      ldv(x + t * C + v * V, a); ldv(gy + t * C + v * V, g); ldv(gamma + v * V, ga);
#pragma unroll
      for (int i = 0; i < V; ++i) o[i] = r * (g[i] * ga[i] - m1 - (a[i] - mu) * r * m2);
      if (add) {
        float e[V];
        ldv(add + t * C + v * V, e);
#pragma unroll
        for (int i = 0; i < V; ++i) o[i] += e[i];
      }
      if (acc) {
        float f[V];
        ldv(gx + t * C + v * V, f);
#pragma unroll
        for (int i = 0; i < V; ++i) o[i] += f[i];
      }
      stv(gx + t * C + v * V, o);
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < C; i += blockDim.x) {
    atomicAdd(dgamma + i, sm[i]);
    atomicAdd(dbeta + i, sm[C + i]);
  }
}

__device__ __forceinline__ float gelu_f(float v) { return 0.5f * v * (1.0f + erff(v * 0.70710678118654752f)); }
__device__ __forceinline__ float gelu_grad_f(float v) {
  return 0.5f * (1.0f + erff(v * 0.70710678118654752f)) + v * __expf(-0.5f * v * v) * 0.39894228040143268f;
}

// bwd == 0: y = GELU(x); bwd == 1: y = g * GELU'(x)
template <typename T>
__global__ void gelu_k(const T* __restrict__ x, const T* __restrict__ g, T* __restrict__ y, size_t nvec, int bwd) {
  constexpr int V = Vec<T>::N;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
    float a[V];
    ldv(x + i * V, a);
    if (bwd) {
      float b[V];
      ldv(g + i * V, b);
#pragma unroll
      for (int k = 0; k < V; ++k) a[k] = b[k] * gelu_grad_f(a[k]);
    } else {
#pragma unroll
      for (int k = 0; k < V; ++k) a[k] = gelu_f(a[k]);
    }
    stv(y + i * V, a);
  }
}

unsigned ln_grid(size_t tokens) {
  const size_t want = (tokens + LN_WARPS - 1) / LN_WARPS;
  return (unsigned)(want < 4 * 148 ? (want ? want : 1) : 4 * 148);
}

}  // namespace

int layernorm_fwd(int dt, const void* x, size_t tokens, int C, float eps, const void* gamma, const void* beta, float* stat,
                  void* y, cudaStream_t st) {
  if (dt == DT_F32) ln_fwd_k<float><<<ln_grid(tokens), LN_WARPS * 32, 0, st>>>((const float*)x, C, tokens, eps, (const float*)gamma, (const float*)beta, stat, (float*)y);
  else ln_fwd_k<bf16><<<ln_grid(tokens), LN_WARPS * 32, 0, st>>>((const bf16*)x, C, tokens, eps, (const bf16*)gamma, (const bf16*)beta, stat, (bf16*)y);
  return 1;
}
int layernorm_bwd(int dt, const void* g_y, const void* x, size_t tokens, int C, const void* gamma, const float* stat,
                  const void* add, void* g_x, int acc, float* dgamma, float* dbeta, cudaStream_t st) {
  const size_t sm = (size_t)2 * C * sizeof(float);
  if (dt == DT_F32) ln_bwd_k<float><<<ln_grid(tokens), LN_WARPS * 32, sm, st>>>((const float*)g_y, (const float*)x, C, tokens, (const float*)gamma, stat, (const float*)add, (float*)g_x, acc, dgamma, dbeta);
  else ln_bwd_k<bf16><<<ln_grid(tokens), LN_WARPS * 32, sm, st>>>((const bf16*)g_y, (const bf16*)x, C, tokens, (const bf16*)gamma, stat, (const bf16*)add, (bf16*)g_x, acc, dgamma, dbeta);
  return 1;
}
int gelu_fwd(int dt, const void* x, void* y, size_t numel, cudaStream_t st) {
  const size_t nvec = numel / (dt == DT_F32 ? 4 : 8);
  const unsigned grid = (unsigned)((nvec + 255) / 256 < 8 * 148 ? (nvec + 255) / 256 : 8 * 148);
  if (dt == DT_F32) gelu_k<float><<<grid ? grid : 1, 256, 0, st>>>((const float*)x, nullptr, (float*)y, nvec, 0);
  else gelu_k<bf16><<<grid ? grid : 1, 256, 0, st>>>((const bf16*)x, nullptr, (bf16*)y, nvec, 0);
  return 1;
}
int gelu_bwd(int dt, const void* x, const void* g, void* g_x, size_t numel, cudaStream_t st) {
  const size_t nvec = numel / (dt == DT_F32 ? 4 : 8);
  const unsigned grid = (unsigned)((nvec + 255) / 256 < 8 * 148 ? (nvec + 255) / 256 : 8 * 148);
  if (dt == DT_F32) gelu_k<float><<<grid ? grid : 1, 256, 0, st>>>((const float*)x, (const float*)g, (float*)g_x, nvec, 1);
  else gelu_k<bf16><<<grid ? grid : 1, 256, 0, st>>>((const bf16*)x, (const bf16*)g, (bf16*)g_x, nvec, 1);
  return 1;
}

}  // namespace pulse

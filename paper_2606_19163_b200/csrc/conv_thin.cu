// conv_thin.cu - 3x3 stride-1 convolutions with 4 channels on one side: the edge convs of the full UNet
// (conv_in 4 -> 320 and the head 320 -> 4, configs[3], configs[4]) and their input / weight gradients.
// They hold 0.02 % of the FLOPs but do not map onto 64-channel TMA boxes; on the generic CUDA-core tile kernel
// (conv_simt.cu, 64 x 64 tiles) the 4-wide side wastes 15/16 of every tile and they cost 17-20 % of a config-4/5
// step.  These kernels are HBM-bound by the wide tensor (21 MB at N = 8, 64 x 64): one pass over it.
//   thin_in   out[p, co]  = b[co] + sum_{tap, c<4} W[co][tap][c] in[p + tap, c]      (conv_in fprop, head dgrad)
//   thin_out  out[p, co<4] = b[co] + sum_{tap, c}  W[co][tap][c] in[p + tap, c]      (head fprop, conv_in dgrad)
//   thin_in_wgrad   dW[co][tap][c<4] += sum_p g[p, co] in[p + tap, c]                (conv_in)
//   thin_out_wgrad  dW[co<4][tap][c] += sum_p g[p, co] in[p + tap, c]                (head)
// SURVEY 8c item 2; dgrad runs as a conv with the flipped / transposed weights like everywhere else.
#include <cstdlib>

#include "common.cuh"
#include "kernels.h"

namespace pulse {

namespace {

constexpr int TC = 4;       // the thin side

// ------------------------------------------------------------------------------ thin input (4 -> cout)
// block: 256 threads = 256 output channels (blockIdx.y selects the chunk); strip = R rows of one image.
// The input patch ((R+2) x (w+2) pixels x 4 channels, fp32, zero padded) sits in shared memory and every tap is
// one broadcast LDS.128; a thread keeps its 36 weights in registers.
template <typename T>
__global__ void __launch_bounds__(256) thin_in_k(const T* __restrict__ in, const T* __restrict__ w,
                                                 const T* __restrict__ bias, T* __restrict__ out, int n, int h, int wd,
                                                 int cout, int R, int accumulate) {
  extern __shared__ float4 patch[];      // [(R+2)][(wd+2)]
  const int strips_per_img = (h + R - 1) / R;
  const int img = blockIdx.x / strips_per_img, y0 = (blockIdx.x % strips_per_img) * R;
  const int pw = wd + 2;
  for (int i = threadIdx.x; i < (R + 2) * pw; i += blockDim.x) {
    const int py = i / pw, px = i - py * pw;
    const int y = y0 + py - 1, x = px - 1;
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (y >= 0 && y < h && x >= 0 && x < wd) {
      const T* p = in + (((size_t)img * h + y) * wd + x) * TC;
      v = make_float4(to_f(p[0]), to_f(p[1]), to_f(p[2]), to_f(p[3]));
    }
    patch[i] = v;
  }
  const int co = blockIdx.y * blockDim.x + threadIdx.x;
  float wr[9][TC];
  float b = 0.f;
  if (co < cout) {
#pragma unroll
    for (int t = 0; t < 9; ++t)
#pragma unroll
      for (int c = 0; c < TC; ++c) wr[t][c] = to_f(w[((size_t)co * 9 + t) * TC + c]);
    if (bias) b = to_f(bias[co]);
  }
  __syncthreads();
  if (co >= cout) return;
  const int rows = min(R, h - y0);
  for (int ry = 0; ry < rows; ++ry)
    for (int x = 0; x < wd; ++x) {
      float acc = b;
#pragma unroll
      for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int s = 0; s < 3; ++s) {
          const float4 v = patch[(ry + r) * pw + x + s];
          acc = fmaf(wr[r * 3 + s][0], v.x, acc); acc = fmaf(wr[r * 3 + s][1], v.y, acc);
          acc = fmaf(wr[r * 3 + s][2], v.z, acc); acc = fmaf(wr[r * 3 + s][3], v.w, acc);
        }
      T* o = out + (((size_t)img * h + y0 + ry) * wd + x) * cout + co;
      if (accumulate) acc += to_f(*o);
      *o = from_f<T>(acc);
    }
}

// dW[co][tap][c] += sum over the strip of g[p, co] in[p + tap, c]; same layout as thin_in_k
template <typename T>
__global__ void __launch_bounds__(256) thin_in_wgrad_k(const T* __restrict__ in, const T* __restrict__ g,
                                                       float* __restrict__ dw, int n, int h, int wd, int cout, int R) {
  extern __shared__ float4 patch[];
  const int strips_per_img = (h + R - 1) / R;
  const int img = blockIdx.x / strips_per_img, y0 = (blockIdx.x % strips_per_img) * R;
  const int pw = wd + 2;
  for (int i = threadIdx.x; i < (R + 2) * pw; i += blockDim.x) {
    const int py = i / pw, px = i - py * pw;
    const int y = y0 + py - 1, x = px - 1;
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (y >= 0 && y < h && x >= 0 && x < wd) {
      const T* p = in + (((size_t)img * h + y) * wd + x) * TC;
      v = make_float4(to_f(p[0]), to_f(p[1]), to_f(p[2]), to_f(p[3]));
    }
    patch[i] = v;
  }
  __syncthreads();
  const int co = blockIdx.y * blockDim.x + threadIdx.x;
  if (co >= cout) return;
  float acc[9][TC];
#pragma unroll
  for (int t = 0; t < 9; ++t)
#pragma unroll
    for (int c = 0; c < TC; ++c) acc[t][c] = 0.f;
  const int rows = min(R, h - y0);
  for (int ry = 0; ry < rows; ++ry)
    for (int x0 = 0; x0 < wd; x0 += 4) {            // 4 pixels per iteration: their g loads are independent
      float gv[4];
#pragma unroll
      for (int u = 0; u < 4; ++u)
        gv[u] = x0 + u < wd ? to_f(g[(((size_t)img * h + y0 + ry) * wd + x0 + u) * cout + co]) : 0.f;
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int x = min(x0 + u, wd - 1);
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
          for (int s = 0; s < 3; ++s) {
            const float4 v = patch[(ry + r) * pw + x + s];
            acc[r * 3 + s][0] = fmaf(gv[u], v.x, acc[r * 3 + s][0]); acc[r * 3 + s][1] = fmaf(gv[u], v.y, acc[r * 3 + s][1]);
            acc[r * 3 + s][2] = fmaf(gv[u], v.z, acc[r * 3 + s][2]); acc[r * 3 + s][3] = fmaf(gv[u], v.w, acc[r * 3 + s][3]);
          }
      }
    }
#pragma unroll
  for (int t = 0; t < 9; ++t)
#pragma unroll
    for (int c = 0; c < TC; ++c) atomicAdd(dw + ((size_t)co * 9 + t) * TC + c, acc[t][c]);
}

// ------------------------------------------------------------------------------ thin output (C -> 4)
// block: PB pixels x (C/8) threads; a thread owns 8 consecutive input channels (one 16-byte load per tap), the
// weights [4][9][C] sit in shared memory as fp32; the PB x (C/8) partial sums are reduced through shared memory.
// Blocks walk pixel groups with a grid stride so that the 46 KB of weights are staged once per block.
template <typename T>
__global__ void __launch_bounds__(512, 2) thin_out_k(const T* __restrict__ in, const T* __restrict__ w,
                                                  const T* __restrict__ bias, T* __restrict__ out, int n, int h, int wd,
                                                  int C, int PB, int accumulate) {
  constexpr int V = Vec<T>::N;
  extern __shared__ float sw[];                  // weights [9][tpp][4 co][V] (+4 floats of padding per thread slot:
                                                 // 16-byte reads at a 144-byte lane stride are bank-conflict free),
                                                 // then [PB][tpp][4] partials
  const int tpp = C / V;                          // threads per pixel
  constexpr int SLOT = TC * V + 4;
  float* red = sw + 9 * tpp * SLOT;
  for (int i = threadIdx.x; i < TC * 9 * C; i += blockDim.x) {
    const int co = i / (9 * C), rem = i - co * 9 * C, tap = rem / C, c = rem - tap * C;
    sw[(tap * tpp + c / V) * SLOT + co * V + (c % V)] = to_f(w[i]);
  }
  __syncthreads();
  const int pl = threadIdx.x / tpp, cv = threadIdx.x - pl * tpp, ch = cv * V;
  const long long M = (long long)n * h * wd;
  for (long long p0 = (long long)blockIdx.x * PB; p0 < M; p0 += (long long)gridDim.x * PB) {
    const long long p = p0 + pl;
    float acc[TC] = {0.f, 0.f, 0.f, 0.f};
    if (p < M) {
      const int x = (int)(p % wd);
      const long long t = p / wd;
      const int y = (int)(t % h);
      const long long img = t / h;
#pragma unroll
      for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int s = 0; s < 3; ++s) {
          const int iy = y + r - 1, ix = x + s - 1;
          if (iy < 0 || iy >= h || ix < 0 || ix >= wd) continue;
          float v[V];
          ldv(in + ((img * h + iy) * wd + ix) * C + ch, v);
          const float4* wp = reinterpret_cast<const float4*>(sw + ((r * 3 + s) * tpp + cv) * SLOT);
#pragma unroll
          for (int co = 0; co < TC; ++co)
#pragma unroll
            for (int q = 0; q < V / 4; ++q) {
              const float4 wv = wp[co * (V / 4) + q];
              acc[co] = fmaf(wv.x, v[4 * q], acc[co]); acc[co] = fmaf(wv.y, v[4 * q + 1], acc[co]);
              acc[co] = fmaf(wv.z, v[4 * q + 2], acc[co]); acc[co] = fmaf(wv.w, v[4 * q + 3], acc[co]);
            }
        }
    }
    *reinterpret_cast<float4*>(red + ((size_t)pl * tpp + cv) * TC) = make_float4(acc[0], acc[1], acc[2], acc[3]);
    __syncthreads();
    if (threadIdx.x < PB * TC) {
      const int q = threadIdx.x / TC, co = threadIdx.x - q * TC;
      const long long pq = p0 + q;
      if (pq < M) {
        float s = bias ? to_f(bias[co]) : 0.f;
        for (int j = 0; j < tpp; ++j) s += red[((size_t)q * tpp + j) * TC + co];
        T* o = out + pq * TC + co;
        if (accumulate) s += to_f(*o);
        *o = from_f<T>(s);
      }
    }
    __syncthreads();
  }
}

// dW[co<4][tap][c] += sum_p g[p, co] in[p + tap, c]: a thread owns (tap, 8 channels) and 4 x 8 accumulators; the
// block walks a contiguous strip of pixels; g of the strip is staged in shared memory.
template <typename T>
__global__ void __launch_bounds__(512, 2) thin_out_wgrad_k(const T* __restrict__ in, const T* __restrict__ g,
                                                        float* __restrict__ dw, int n, int h, int wd, int C,
                                                        int strip) {
  constexpr int V = Vec<T>::N;
  extern __shared__ float sg[];                  // [strip][4]
  const int tpp = C / V;
  const int tap = threadIdx.x / tpp, cv = threadIdx.x - tap * tpp, ch = cv * V;
  const int r = tap / 3, s = tap - r * 3;
  const long long M = (long long)n * h * wd;
  const long long pb = (long long)blockIdx.x * strip, pe = pb + strip < M ? pb + strip : M;
  for (int i = threadIdx.x; i < (int)(pe - pb) * TC; i += blockDim.x) sg[i] = to_f(g[pb * TC + i]);
  __syncthreads();
  if (tap >= 9) return;
  float acc[TC][V];
#pragma unroll
  for (int co = 0; co < TC; ++co)
#pragma unroll
    for (int i = 0; i < V; ++i) acc[co][i] = 0.f;
  int x = (int)(pb % wd);
  long long t = pb / wd;
  int y = (int)(t % h);
  long long img = t / h;
  for (long long p = pb; p < pe; p += 4) {          // 4 pixels per iteration: their loads are independent
    float v[4][V];
    bool ok[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int iy = y + r - 1, ix = x + s - 1;
      ok[u] = p + u < pe && iy >= 0 && iy < h && ix >= 0 && ix < wd;
      if (ok[u]) ldv(in + ((img * h + iy) * wd + ix) * C + ch, v[u]);
      if (++x == wd) { x = 0; if (++y == h) { y = 0; ++img; } }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      if (!ok[u]) continue;
      const float4 gv = *reinterpret_cast<const float4*>(sg + (p + u - pb) * TC);
#pragma unroll
      for (int i = 0; i < V; ++i) {
        acc[0][i] = fmaf(gv.x, v[u][i], acc[0][i]); acc[1][i] = fmaf(gv.y, v[u][i], acc[1][i]);
        acc[2][i] = fmaf(gv.z, v[u][i], acc[2][i]); acc[3][i] = fmaf(gv.w, v[u][i], acc[3][i]);
      }
    }
  }
#pragma unroll
  for (int co = 0; co < TC; ++co)
#pragma unroll
    for (int i = 0; i < V; ++i) atomicAdd(dw + ((size_t)co * 9 + tap) * C + ch + i, acc[co][i]);
}

template <typename K> void big_smem(K kernel, size_t bytes) {
  if (bytes > 48 * 1024) cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

}  // namespace

// ------------------------------------------------------------------------------ dispatch
static bool thin_common(int ksize, int stride, int mode, const Cat& src, int hin, int win, int hout, int wout) {
  return ksize == 3 && stride == 1 && mode == CONV_FPROP && src.c1 == 0 && hin == hout && win == wout;
}
bool conv_thin_supported(const ConvArgs& a) {
  if (!thin_common(a.ksize, a.stride, a.mode, a.src, a.hin, a.win, a.hout, a.wout) || a.pn || a.residual) return false;
  const int vec = a.dt == DT_F32 ? 4 : 8;
  if (a.src.c0 == TC && a.cout >= 32) return (size_t)3 * (a.win + 2) * 16 <= 96 * 1024;
  if (a.cout == TC && a.src.c0 % vec == 0 && a.src.c0 / vec <= 64) return true;
  return false;
}
int conv_thin(const ConvArgs& a, cudaStream_t st) {
  if (a.src.c0 == TC) {
    int R = 128 / a.win; if (R < 1) R = 1; if (R > a.hin) R = a.hin;
    const int chunks = (a.cout + 255) / 256;
    int threads = ((a.cout + chunks - 1) / chunks + 31) / 32 * 32;
    dim3 grid(a.n * ((a.hin + R - 1) / R), (a.cout + threads - 1) / threads);
    const size_t sm = (size_t)(R + 2) * (a.win + 2) * sizeof(float4);
    if (a.dt == DT_F32) {
      big_smem(thin_in_k<float>, sm);
      thin_in_k<float><<<grid, threads, sm, st>>>((const float*)a.src.p0, (const float*)a.w, (const float*)a.bias,
                                                  (float*)a.out, a.n, a.hin, a.win, a.cout, R, a.accumulate);
    } else {
      big_smem(thin_in_k<bf16>, sm);
      thin_in_k<bf16><<<grid, threads, sm, st>>>((const bf16*)a.src.p0, (const bf16*)a.w, (const bf16*)a.bias,
                                                 (bf16*)a.out, a.n, a.hin, a.win, a.cout, R, a.accumulate);
    }
    return 1;
  }
  const int vec = a.dt == DT_F32 ? 4 : 8, C = a.src.c0, tpp = C / vec;
  int PB = 512 / tpp; if (PB < 1) PB = 1;
  const int threads = PB * tpp;
  const long long M = (long long)a.n * a.hin * a.win;
  long long blocks = (M + PB - 1) / PB;
  if (blocks > 296) blocks = 296;
  const size_t sm = ((size_t)9 * tpp * (TC * vec + 4) + (size_t)PB * tpp * TC) * sizeof(float);
  if (a.dt == DT_F32) {
    big_smem(thin_out_k<float>, sm);
    thin_out_k<float><<<(unsigned)blocks, threads, sm, st>>>((const float*)a.src.p0, (const float*)a.w,
                                                             (const float*)a.bias, (float*)a.out, a.n, a.hin, a.win, C,
                                                             PB, a.accumulate);
  } else {
    big_smem(thin_out_k<bf16>, sm);
    thin_out_k<bf16><<<(unsigned)blocks, threads, sm, st>>>((const bf16*)a.src.p0, (const bf16*)a.w, (const bf16*)a.bias,
                                                            (bf16*)a.out, a.n, a.hin, a.win, C, PB, a.accumulate);
  }
  return 1;
}

bool wgrad_thin_supported(const WgradArgs& a) {
  if (!thin_common(a.ksize, a.stride, CONV_FPROP, a.src, a.hin, a.win, a.hout, a.wout)) return false;
  const int vec = a.dt == DT_F32 ? 4 : 8;
  if (a.src.c0 == TC && a.cout >= 32) return (size_t)3 * (a.win + 2) * 16 <= 96 * 1024;
  if (a.cout == TC && a.src.c0 % vec == 0 && 9 * (a.src.c0 / vec) <= 512) return true;
  return false;
}
int wgrad_thin(const WgradArgs& a, cudaStream_t st) {
  if (a.src.c0 == TC) {
    int R = 128 / a.win; if (R < 1) R = 1; if (R > a.hin) R = a.hin;
    const int chunks = (a.cout + 255) / 256;
    int threads = ((a.cout + chunks - 1) / chunks + 31) / 32 * 32;
    dim3 grid(a.n * ((a.hin + R - 1) / R), (a.cout + threads - 1) / threads);
    const size_t sm = (size_t)(R + 2) * (a.win + 2) * sizeof(float4);
    if (a.dt == DT_F32) {
      big_smem(thin_in_wgrad_k<float>, sm);
      thin_in_wgrad_k<float><<<grid, threads, sm, st>>>((const float*)a.src.p0, (const float*)a.g, a.dw, a.n, a.hin, a.win,
                                                        a.cout, R);
    } else {
      big_smem(thin_in_wgrad_k<bf16>, sm);
      thin_in_wgrad_k<bf16><<<grid, threads, sm, st>>>((const bf16*)a.src.p0, (const bf16*)a.g, a.dw, a.n, a.hin, a.win,
                                                       a.cout, R);
    }
    return 1;
  }
  const int vec = a.dt == DT_F32 ? 4 : 8, C = a.src.c0, tpp = C / vec;
  const int threads = (9 * tpp + 31) / 32 * 32;
  const long long M = (long long)a.n * a.hin * a.win;
  int strip = (int)((M + 295) / 296);               // ~2 blocks per SM: fewer, longer strips = fewer atomics
  if (strip < 16) strip = 16;
  if (strip > 2048) strip = 2048;
  const long long blocks = (M + strip - 1) / strip;
  const size_t sm = (size_t)strip * TC * sizeof(float);
  if (a.dt == DT_F32)
    thin_out_wgrad_k<float><<<(unsigned)blocks, threads, sm, st>>>((const float*)a.src.p0, (const float*)a.g, a.dw, a.n,
                                                                   a.hin, a.win, C, strip);
  else
    thin_out_wgrad_k<bf16><<<(unsigned)blocks, threads, sm, st>>>((const bf16*)a.src.p0, (const bf16*)a.g, a.dw, a.n,
                                                                  a.hin, a.win, C, strip);
  return 1;
}

}  // namespace pulse

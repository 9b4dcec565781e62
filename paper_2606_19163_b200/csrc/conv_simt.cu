// conv_simt.cu - CUDA-core implicit-GEMM convolution (fp32 accumulate), any shape.
// Role: (1) the fp32 debug path of configs[0] (north_star: "<= 1e-4 relative for an
// fp32 debug path"; tcgen05 kind::tf32 has a 10-bit mantissa and cannot meet it),
// (2) the edge convs with Cin = 4 / Cout = 4 (0.02 % of FLOPs) that do not map onto
// 64-channel TMA boxes, (3) PULSE_FLAG_FORCE_SIMT on-device cross-check of the tensor
// core path.  SURVEY 8c item 2:
//   out[n,y,x,co] = b[co] + sum_{r,s,ci} W[co][r][s][ci] in[n, y st + r - pad, x st + s - pad, ci]
#include <cstdlib>

#include "common.cuh"
#include "kernels.h"

namespace pulse {

namespace {
constexpr int TM = 64, TN = 64, TK = 16;

struct SimtP {
  const void* p0; int c0; const void* p1; int c1;
  int n, hin, win, hout, wout, ksize, stride, mode, cout;
  const void* w; const void* bias; const float* pn; const void* residual; void* out; int accumulate;
};

template <typename T>
__global__ void __launch_bounds__(256) conv_simt_k(SimtP a) {
  __shared__ float sA[TK][TM + 4];
  __shared__ float sB[TK][TN + 4];
  __shared__ int spn[TM], spy[TM], spx[TM];
  const int tid = threadIdx.x;
  const int ctot = a.c0 + a.c1, K = a.ksize * a.ksize * ctot, pad = (a.ksize - 1) / 2;
  const long long M = (long long)a.n * a.hout * a.wout;
  const long long m0 = (long long)blockIdx.x * TM;
  const int co0 = blockIdx.y * TN;
  if (tid < TM) {
    long long m = m0 + tid;
    if (m < M) {
      spx[tid] = (int)(m % a.wout);
      long long t = m / a.wout;
      spy[tid] = (int)(t % a.hout);
      spn[tid] = (int)(t / a.hout);
    } else {
      spn[tid] = -1; spy[tid] = 0; spx[tid] = 0;
    }
  }
  __syncthreads();
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;
  const int lp = tid >> 2, lk = (tid & 3) * 4;     // loader role: row (pixel / cout) and 4 consecutive k
  const int ty = tid >> 4, tx = tid & 15;          // compute role
  const T* w = (const T*)a.w;
  for (int k0 = 0; k0 < K; k0 += TK) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int k = k0 + lk + j;
      float va = 0.f, vb = 0.f;
      if (k < K) {
        const int tap = k / ctot, c = k - tap * ctot;
        const int r = tap / a.ksize, s = tap - r * a.ksize;
        const int nn = spn[lp];
        if (nn >= 0) {
          int ty_ = spy[lp] * (a.mode == CONV_FPROP ? a.stride : 1) + r - pad;
          int tx_ = spx[lp] * (a.mode == CONV_FPROP ? a.stride : 1) + s - pad;
          bool ok = ty_ >= 0 && tx_ >= 0;
          if (a.mode == CONV_DGRAD_S2) {
            ok = ok && !(ty_ & 1) && !(tx_ & 1);
            ty_ >>= 1; tx_ >>= 1;
          }
          ok = ok && ty_ < a.hin && tx_ < a.win;
          if (ok) {
            const size_t pix = ((size_t)nn * a.hin + ty_) * a.win + tx_;
            va = c < a.c0 ? to_f(((const T*)a.p0)[pix * a.c0 + c]) : to_f(((const T*)a.p1)[pix * a.c1 + (c - a.c0)]);
          }
        }
        const int co = co0 + lp;
        if (co < a.cout) vb = to_f(w[(size_t)co * K + k]);
      }
      sA[lk + j][lp] = va;
      sB[lk + j][lp] = vb;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < TK; ++kk) {
      float av[4], bv[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) { av[i] = sA[kk][ty * 4 + i]; bv[i] = sB[kk][tx * 4 + i]; }
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
    }
    __syncthreads();
  }
  T* out = (T*)a.out;
  const T* res = (const T*)a.residual;
  const T* bias = (const T*)a.bias;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int pl = ty * 4 + i;
    const int nn = spn[pl];
    if (nn < 0) continue;
    const size_t m = (size_t)(m0 + pl);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int co = co0 + tx * 4 + j;
      if (co >= a.cout) continue;
      float v = acc[i][j];
      if (bias) v += to_f(bias[co]);
      if (a.pn) v += a.pn[(size_t)nn * a.cout + co];
      if (res) v += to_f(res[m * a.cout + co]);
      if (a.accumulate) v += to_f(out[m * a.cout + co]);
      out[m * a.cout + co] = from_f<T>(v);
    }
  }
}

struct WgP {
  const void* p0; int c0; const void* p1; int c1;
  int n, hin, win, hout, wout, ksize, stride, cout;
  const void* g; float* dw; int pix_per_split;
};

template <typename T>
__global__ void __launch_bounds__(256) wgrad_simt_k(WgP a) {
  __shared__ float sA[TK][TM + 4];     // [pixel][co]
  __shared__ float sB[TK][TN + 4];     // [pixel][kidx]
  const int tid = threadIdx.x;
  const int ctot = a.c0 + a.c1, K = a.ksize * a.ksize * ctot, pad = (a.ksize - 1) / 2;
  const long long M = (long long)a.n * a.hout * a.wout;
  const int co0 = blockIdx.x * TM, k0 = blockIdx.y * TN;
  const long long pb = (long long)blockIdx.z * a.pix_per_split;
  const long long pe = pb + a.pix_per_split < M ? pb + a.pix_per_split : M;
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;
  const int lpix = tid >> 4, lcol = (tid & 15) * 4;    // loader: pixel row, 4 consecutive columns
  const int ty = tid >> 4, tx = tid & 15;
  const T* g = (const T*)a.g;
  for (long long p0 = pb; p0 < pe; p0 += TK) {
    const long long m = p0 + lpix;
    const bool live = m < pe;
    int nn = 0, y = 0, x = 0;
    if (live) {
      x = (int)(m % a.wout);
      long long t = m / a.wout;
      y = (int)(t % a.hout);
      nn = (int)(t / a.hout);
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      float va = 0.f, vb = 0.f;
      if (live) {
        const int co = co0 + lcol + j;
        if (co < a.cout) va = to_f(g[(size_t)m * a.cout + co]);
        const int k = k0 + lcol + j;
        if (k < K) {
          const int tap = k / ctot, c = k - tap * ctot;
          const int r = tap / a.ksize, s = tap - r * a.ksize;
          const int iy = y * a.stride + r - pad, ix = x * a.stride + s - pad;
          if (iy >= 0 && ix >= 0 && iy < a.hin && ix < a.win) {
            const size_t pix = ((size_t)nn * a.hin + iy) * a.win + ix;
            vb = c < a.c0 ? to_f(((const T*)a.p0)[pix * a.c0 + c]) : to_f(((const T*)a.p1)[pix * a.c1 + (c - a.c0)]);
          }
        }
      }
      sA[lpix][lcol + j] = va;
      sB[lpix][lcol + j] = vb;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < TK; ++kk) {
      float av[4], bv[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) { av[i] = sA[kk][ty * 4 + i]; bv[i] = sB[kk][tx * 4 + i]; }
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int co = co0 + ty * 4 + i;
    if (co >= a.cout) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int k = k0 + tx * 4 + j;
      if (k < K) atomicAdd(a.dw + (size_t)co * K + k, acc[i][j]);
    }
  }
}
}  // namespace

int conv_simt(const ConvArgs& a, cudaStream_t st) {
  if (conv_thin_supported(a)) return conv_thin(a, st);
  SimtP p;
  p.p0 = a.src.p0; p.c0 = a.src.c0; p.p1 = a.src.p1; p.c1 = a.src.c1;
  p.n = a.n; p.hin = a.hin; p.win = a.win; p.hout = a.hout; p.wout = a.wout;
  p.ksize = a.ksize; p.stride = a.stride; p.mode = a.mode; p.cout = a.cout;
  p.w = a.w; p.bias = a.bias; p.pn = a.pn; p.residual = a.residual; p.out = a.out; p.accumulate = a.accumulate;
  const long long M = (long long)a.n * a.hout * a.wout;
  dim3 grid((unsigned)((M + TM - 1) / TM), (a.cout + TN - 1) / TN);
  if (a.dt == DT_F32) conv_simt_k<float><<<grid, 256, 0, st>>>(p);
  else conv_simt_k<bf16><<<grid, 256, 0, st>>>(p);
  return 1;
}

int wgrad_simt(const WgradArgs& a, cudaStream_t st) {
  if (wgrad_thin_supported(a)) return wgrad_thin(a, st);
  WgP p;
  p.p0 = a.src.p0; p.c0 = a.src.c0; p.p1 = a.src.p1; p.c1 = a.src.c1;
  p.n = a.n; p.hin = a.hin; p.win = a.win; p.hout = a.hout; p.wout = a.wout;
  p.ksize = a.ksize; p.stride = a.stride; p.cout = a.cout; p.g = a.g; p.dw = a.dw;
  const int K = a.ksize * a.ksize * a.src.c();
  const long long M = (long long)a.n * a.hout * a.wout;
  const int tiles = ((a.cout + TM - 1) / TM) * ((K + TN - 1) / TN);
  int splits = (592 + tiles - 1) / tiles;
  const long long maxs = (M + 4 * TK - 1) / (4 * TK);
  if (splits > maxs) splits = (int)maxs;
  if (splits < 1) splits = 1;
  long long pps = (M + splits - 1) / splits;
  pps = (pps + TK - 1) / TK * TK;
  splits = (int)((M + pps - 1) / pps);
  p.pix_per_split = (int)pps;
  dim3 grid((a.cout + TM - 1) / TM, (K + TN - 1) / TN, splits);
  if (a.dt == DT_F32) wgrad_simt_k<float><<<grid, 256, 0, st>>>(p);
  else wgrad_simt_k<bf16><<<grid, 256, 0, st>>>(p);
  return 1;
}

}  // namespace pulse

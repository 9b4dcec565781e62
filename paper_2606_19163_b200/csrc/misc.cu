// misc.cu - the small, HBM- or latency-bound ops of the stage: per-channel pixel sums
// (bias / temb-projection gradients), the [N<=16, <=1280] linears of the timestep path,
// sinusoidal embedding, MSE loss+gradient, nearest-2x upsample and its adjoint, in-place
// add, and the weight flip/transpose that turns dgrad into fprop.
#include "common.cuh"
#include "kernels.h"

namespace pulse {

// ------------------------------------------------------------------ column sums over pixels
// cs[n][c] += sum_pix g[n][pix][c].  Only for gradient tensors whose writers could not emit their own column
// sums (the loss gradient that enters from outside, conv-dgrad outputs); everything written by the GroupNorm
// backward carries its sums already (norm.cu).  One fp32 atomic per channel per CTA.
template <typename T>
__global__ void __launch_bounds__(512, 2) colsum_k(const T* __restrict__ g, int hw, int C, float* __restrict__ cs) {
  constexpr int V = Vec<T>::N;
  extern __shared__ float sm[];
  const int n = blockIdx.y, nchunks = gridDim.x;
  const int ppc = (hw + nchunks - 1) / nchunks;
  const int pb = blockIdx.x * ppc, pe = min(hw, pb + ppc);
  const int ch = threadIdx.x * V, rows = blockDim.y, ty = threadIdx.y;
  float s[V];
#pragma unroll
  for (int i = 0; i < V; ++i) s[i] = 0.f;
  for (int p = pb + ty; p < pe; p += 4 * rows) {
    float v[4][V];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      if (p + u * rows < pe) ldv(g + ((size_t)n * hw + p + u * rows) * C + ch, v[u]);
      else {
#pragma unroll
        for (int i = 0; i < V; ++i) v[u][i] = 0.f;
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int i = 0; i < V; ++i) s[i] += v[u][i];
  }
  if (rows == 1) {
#pragma unroll
    for (int i = 0; i < V; ++i) atomicAdd(cs + (size_t)n * C + ch + i, s[i]);
    return;
  }
#pragma unroll
  for (int i = 0; i < V; ++i) sm[ty * C + ch + i] = s[i];
  __syncthreads();
  for (int c = ty * blockDim.x + threadIdx.x; c < C; c += blockDim.x * blockDim.y) {
    float t = 0.f;
    for (int r = 0; r < rows; ++r) t += sm[r * C + c];
    atomicAdd(cs + (size_t)n * C + c, t);
  }
}

// any C (used for Cout = 4): one block per (channel, image)
template <typename T>
__global__ void colsum_scalar_k(const T* __restrict__ g, int hw, int C, float* cs) {
  const int c = blockIdx.x, n = blockIdx.y;
  __shared__ float sh[32];
  float s = 0.f;
  for (int p = threadIdx.x; p < hw; p += blockDim.x) s += to_f(g[((size_t)n * hw + p) * C + c]);
  s = warp_sum(s);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    float v = 0.f;
    for (int i = 0; i < (int)(blockDim.x >> 5); ++i) v += sh[i];
    atomicAdd(cs + (size_t)n * C + c, v);
  }
}

int colsum(int dt, const void* g, int n, int hw, int c, float* cs, cudaStream_t st) {
  const int vec = dt == DT_F32 ? 4 : 8;
  if (c % vec || c / vec > 512) {
    if (dt == DT_F32) colsum_scalar_k<float><<<dim3(c, n), 256, 0, st>>>((const float*)g, hw, c, cs);
    else colsum_scalar_k<bf16><<<dim3(c, n), 256, 0, st>>>((const bf16*)g, hw, c, cs);
    return 1;
  }
  const RowPlan pl = row_plan(dt, hw, c, n, 512);
  dim3 grid(pl.nchunks, n), block(pl.tpr, pl.rows);
  const size_t smem = pl.rows > 1 ? (size_t)pl.rows * c * sizeof(float) : 0;
  if (dt == DT_F32) colsum_k<float><<<grid, block, smem, st>>>((const float*)g, hw, c, cs);
  else colsum_k<bf16><<<grid, block, smem, st>>>((const bf16*)g, hw, c, cs);
  return 1;
}

// ------------------------------------------------------------------ batched per-op small kernels
constexpr int BATCH = 16;
struct ProjBatch { int count; ProjEntry e[BATCH]; };
struct SmallGradBatch { int count; SmallGradEntry e[BATCH]; };
struct TransposeBatch { int count; TransposeEntry e[BATCH]; };

// out[n][o] = sum_j W[o][j] f(in[n][j]) + b[o], f = SiLU or identity, for up to 16 weight matrices in one launch
// (the temb projections of every ResBlock; the two linears of the timestep MLP, row a1).
// Latency-bound GEMVs (n <= 8 rows): a warp owns one output row and requests its first 5 weight vectors (16 bytes
// each) BEFORE the block stages f(in) in shared memory ([n <= 8][din] floats), so that the two global round trips
// overlap; then FMAs against shared memory, a warp reduction per row of in, one store.
constexpr int RD_PRE = 5;         // weight vectors per lane in flight (din <= 1280 for bf16: the whole row)
template <typename T>
__global__ void __launch_bounds__(256) rowdot_k(const float* __restrict__ in, int n0, int nn, int din, int silu_in,
                                                const __grid_constant__ ProjBatch b) {
  constexpr int V = Vec<T>::N;
  extern __shared__ float se[];        // [nn][din]
  const ProjEntry& e = b.e[blockIdx.y];
  const int o0 = blockIdx.x * 8;
  if (o0 >= e.cout) return;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int o = o0 + warp;
  const bool vec_ok = din % V == 0;
  const T* w = (const T*)e.w + (size_t)(o < e.cout ? o : o0) * din;
  const int nvec = din / V;            // vectors per row (vec_ok)
  uint4 pre[RD_PRE];
  if (vec_ok) {
#pragma unroll
    for (int u = 0; u < RD_PRE; ++u) {
      const int v = lane + 32 * u;
      pre[u] = v < nvec ? *reinterpret_cast<const uint4*>(w + (size_t)v * V) : make_uint4(0u, 0u, 0u, 0u);
    }
  }
  if (din % 4 == 0) {                  // stage f(in): float4 loads, all of a thread's requests before the first use
    const int n4 = nn * din / 4;
    const float4* src = reinterpret_cast<const float4*>(in + (size_t)n0 * din);
    for (int i0 = threadIdx.x; i0 < n4; i0 += 4 * 256) {
      float4 t[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) if (i0 + u * 256 < n4) t[u] = src[i0 + u * 256];
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (i0 + u * 256 < n4) {
          if (silu_in) { t[u].x = siluf_(t[u].x); t[u].y = siluf_(t[u].y); t[u].z = siluf_(t[u].z); t[u].w = siluf_(t[u].w); }
          reinterpret_cast<float4*>(se)[i0 + u * 256] = t[u];
        }
    }
  } else {
    for (int i = threadIdx.x; i < nn * din; i += 256) {
      const float t = in[(size_t)n0 * din + i];
      se[i] = silu_in ? siluf_(t) : t;
    }
  }
  __syncthreads();
  if (o >= e.cout) return;
  float acc[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) acc[j] = 0.f;
  if (vec_ok) {
    for (int v0 = 0; v0 < nvec; v0 += 32 * RD_PRE) {
      if (v0) {                          // rows longer than 32 * RD_PRE vectors: next batch
#pragma unroll
        for (int u = 0; u < RD_PRE; ++u) {
          const int v = v0 + lane + 32 * u;
          pre[u] = v < nvec ? *reinterpret_cast<const uint4*>(w + (size_t)v * V) : make_uint4(0u, 0u, 0u, 0u);
        }
      }
#pragma unroll
      for (int u = 0; u < RD_PRE; ++u) {
        const int v = v0 + lane + 32 * u;
        if (v < nvec) {
          float wv[V];
          unpack(pre[u], wv);
#pragma unroll
          for (int j = 0; j < 8; ++j)
            if (j < nn) {
              const float* x = se + j * din + v * V;
#pragma unroll
              for (int k = 0; k < V; k += 4) {
                const float4 xv = *reinterpret_cast<const float4*>(x + k);
                acc[j] = fmaf(wv[k], xv.x, acc[j]); acc[j] = fmaf(wv[k + 1], xv.y, acc[j]);
                acc[j] = fmaf(wv[k + 2], xv.z, acc[j]); acc[j] = fmaf(wv[k + 3], xv.w, acc[j]);
              }
            }
        }
      }
    }
  } else {
    for (int i = lane; i < din; i += 32) {
      const float wv = to_f(w[i]);
#pragma unroll
      for (int j = 0; j < 8; ++j)
        if (j < nn) acc[j] = fmaf(wv, se[j * din + i], acc[j]);
    }
  }
  const float bo = e.b ? to_f(((const T*)e.b)[o]) : 0.f;
#pragma unroll
  for (int j = 0; j < 8; ++j)
    if (j < nn) {
      const float t = warp_sum(acc[j]);
      if (lane == 0) e.out[(size_t)(n0 + j) * e.cout + o] = t + bo;
    }
}

static int rowdot_batch(int dt, const float* in, int n, int din, int silu_in, const ProjEntry* e, int count, cudaStream_t st) {
  int launches = 0;
  for (int i0 = 0; i0 < count; i0 += BATCH) {
    ProjBatch b;
    b.count = count - i0 < BATCH ? count - i0 : BATCH;
    int maxc = 0;
    for (int i = 0; i < b.count; ++i) { b.e[i] = e[i0 + i]; if (e[i0 + i].cout > maxc) maxc = e[i0 + i].cout; }
    for (int n0 = 0; n0 < n; n0 += 8) {
      const int nn = n - n0 < 8 ? n - n0 : 8;
      dim3 grid((maxc + 7) / 8, b.count);
      const size_t smem = (size_t)nn * din * sizeof(float);
      if (dt == DT_F32) rowdot_k<float><<<grid, 256, smem, st>>>(in, n0, nn, din, silu_in, b);
      else rowdot_k<bf16><<<grid, 256, smem, st>>>(in, n0, nn, din, silu_in, b);
      ++launches;
    }
  }
  return launches;
}
int temb_proj_batch(int dt, const float* emb, int n, int T, const ProjEntry* e, int count, cudaStream_t st) {
  return rowdot_batch(dt, emb, n, T, 1, e, count, st);
}

// Per op (blockIdx.z), channel chunk of 32 (blockIdx.y), 256 columns j of the temb dimension (blockIdx.x):
//   dtw[c][j] += sum_n gp[n][c] silu(emb[n][j]);  g_emb[n][j] += silu'(emb[n][j]) sum_c gp[n][c] tw[c][j];
//   blockIdx.x == 0 also folds the bias gradients: db_out (+ db_out2) += sum_n cs_out, db1 / dtb += sum_n gp.
template <typename T>
__global__ void __launch_bounds__(256) small_grads_k(const float* __restrict__ emb, float* g_emb, int n, int Tdim,
                                                     const __grid_constant__ SmallGradBatch b) {
  const SmallGradEntry& e = b.e[blockIdx.z];
  const int c0 = blockIdx.y * 32;
  if (c0 >= e.cout) return;
  const int cn = min(32, e.cout - c0);
  __shared__ float sgp[8][32];
  if (blockIdx.x == 0 && threadIdx.x < cn) {
    const int c = c0 + threadIdx.x;
    float s = 0.f, t = 0.f;
    for (int j = 0; j < n; ++j) {
      s += e.cs_out[(size_t)j * e.cout + c];
      if (e.gp) t += e.gp[(size_t)j * e.cout + c];
    }
    e.db_out[c] += s;
    if (e.db_out2) e.db_out2[c] += s;
    if (e.gp) { e.db1[c] += t; e.dtb[c] += t; }
  }
  if (!e.gp) return;
  const int j = blockIdx.x * 256 + threadIdx.x;
  const T* tw = (const T*)e.tw;
  for (int n0 = 0; n0 < n; n0 += 8) {
    const int nn = min(8, n - n0);
    __syncthreads();
    {   // all 8 x 32 entries are written: rows >= nn must be 0, not stale shared memory (0 x NaN = NaN)
      const int r = threadIdx.x >> 5, c = threadIdx.x & 31;
      sgp[r][c] = (r < nn && c < cn) ? e.gp[(size_t)(n0 + r) * e.cout + c0 + c] : 0.f;
    }
    __syncthreads();
    if (j < Tdim) {
      float se[8], ge[8];
#pragma unroll
      for (int r = 0; r < 8; ++r) { se[r] = r < nn ? siluf_(emb[(size_t)(n0 + r) * Tdim + j]) : 0.f; ge[r] = 0.f; }
      for (int cb = 0; cb < cn; cb += 8) {            // 8 channels per batch: 16 independent loads in flight
        float w[8], old[8];
#pragma unroll
        for (int u = 0; u < 8; ++u)
          if (cb + u < cn) {
            w[u] = to_f(tw[(size_t)(c0 + cb + u) * Tdim + j]);
            old[u] = e.dtw[(size_t)(c0 + cb + u) * Tdim + j];
          }
#pragma unroll
        for (int u = 0; u < 8; ++u)
          if (cb + u < cn) {
            const int c = cb + u;
            float d = old[u];
#pragma unroll
            for (int r = 0; r < 8; ++r) { d = fmaf(sgp[r][c], se[r], d); ge[r] = fmaf(sgp[r][c], w[u], ge[r]); }
            e.dtw[(size_t)(c0 + c) * Tdim + j] = d;
          }
      }
      if (g_emb)
#pragma unroll
        for (int r = 0; r < 8; ++r)
          if (r < nn) atomicAdd(g_emb + (size_t)(n0 + r) * Tdim + j, ge[r] * silu_gradf_(emb[(size_t)(n0 + r) * Tdim + j]));
    }
  }
}

int small_grads_batch(int dt, const float* emb, float* g_emb, int n, int T, const SmallGradEntry* e, int count,
                      cudaStream_t st) {
  int launches = 0;
  for (int i0 = 0; i0 < count; i0 += BATCH) {
    SmallGradBatch b;
    b.count = count - i0 < BATCH ? count - i0 : BATCH;
    int maxc = 0;
    for (int i = 0; i < b.count; ++i) { b.e[i] = e[i0 + i]; if (e[i0 + i].cout > maxc) maxc = e[i0 + i].cout; }
    dim3 grid((T + 255) / 256, (maxc + 31) / 32, b.count);
    if (dt == DT_F32) small_grads_k<float><<<grid, 256, 0, st>>>(emb, g_emb, n, T, b);
    else small_grads_k<bf16><<<grid, 256, 0, st>>>(emb, g_emb, n, T, b);
    ++launches;
  }
  return launches;
}

// ------------------------------------------------------------------ tiny linears (timestep path)
int linear_fwd(int dt, const float* in, int n, int din, int dout, const void* w, const void* b, int silu_in,
               float* out, cudaStream_t st) {
  const ProjEntry e{w, b, out, dout};
  return rowdot_batch(dt, in, n, din, silu_in, &e, 1, st);
}

// dW[o][i] += sum_n g[n][o] f(in[n][i]); db[o] += sum_n g[n][o]
__global__ void linear_bwd_w_k(const float* __restrict__ in, const float* __restrict__ g, int n, int din, int dout,
                               int silu_in, float* __restrict__ dw, float* __restrict__ db) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)din * dout) return;
  const int o = idx / din, i = idx % din;
  float s = 0.f, sb = 0.f;
  for (int j = 0; j < n; ++j) {
    float x = in[(size_t)j * din + i];
    if (silu_in) x = siluf_(x);
    const float gv = g[(size_t)j * dout + o];
    s = fmaf(gv, x, s);
    sb += gv;
  }
  dw[idx] += s;
  if (i == 0 && db) db[o] += sb;
}

// g_in[n][i] += (sum_{o in chunk} g[n][o] W[o][i]) f'(in[n][i])   (atomic; caller zeroes g_in when it must not accumulate)
template <typename T>
__global__ void linear_bwd_in_k(const float* __restrict__ in, const float* __restrict__ g, int n, int din, int dout,
                                const T* __restrict__ w, int silu_in, float* __restrict__ g_in, int ochunk) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= din) return;
  const int o0 = blockIdx.z * ochunk, o1 = min(dout, o0 + ochunk);
  float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
  int o = o0;
  for (; o + 4 <= o1; o += 4) {
    s0 = fmaf(g[(size_t)j * dout + o], to_f(w[(size_t)o * din + i]), s0);
    s1 = fmaf(g[(size_t)j * dout + o + 1], to_f(w[(size_t)(o + 1) * din + i]), s1);
    s2 = fmaf(g[(size_t)j * dout + o + 2], to_f(w[(size_t)(o + 2) * din + i]), s2);
    s3 = fmaf(g[(size_t)j * dout + o + 3], to_f(w[(size_t)(o + 3) * din + i]), s3);
  }
  for (; o < o1; ++o) s0 = fmaf(g[(size_t)j * dout + o], to_f(w[(size_t)o * din + i]), s0);
  float s = (s0 + s1) + (s2 + s3);
  if (silu_in) s *= silu_gradf_(in[(size_t)j * din + i]);
  atomicAdd(g_in + (size_t)j * din + i, s);
}

int linear_bwd(int dt, const float* in, const float* g, int n, int din, int dout, const void* w, int silu_in,
               float* dw, float* db, float* g_in, int acc_g_in, cudaStream_t st) {
  int launches = 1;
  const size_t tot = (size_t)din * dout;
  linear_bwd_w_k<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(in, g, n, din, dout, silu_in, dw, db);
  if (g_in) {
    if (!acc_g_in) cudaMemsetAsync(g_in, 0, (size_t)n * din * sizeof(float), st);
    const int ochunk = 32;
    dim3 grid((din + 127) / 128, n, (dout + ochunk - 1) / ochunk);
    if (dt == DT_F32)
      linear_bwd_in_k<float><<<grid, 128, 0, st>>>(in, g, n, din, dout, (const float*)w, silu_in, g_in, ochunk);
    else
      linear_bwd_in_k<bf16><<<grid, 128, 0, st>>>(in, g, n, din, dout, (const bf16*)w, silu_in, g_in, ochunk);
    ++launches;
  }
  return launches;
}

// ------------------------------------------------------------------ sinusoidal embedding
__global__ void sinusoidal_k(const int64_t* __restrict__ t, int n, int d, float* __restrict__ out) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x, half = d / 2;
  if (idx >= n * half) return;
  const int j = idx / half, i = idx % half;
  // f_i = exp(-ln(10000) i / half); angle in double so that t up to 999 keeps fp32-exact phase
  const double f = exp(-9.210340371976184 * (double)i / (double)half);
  const double a = (double)t[j] * f;
  out[(size_t)j * d + i] = (float)cos(a);
  out[(size_t)j * d + half + i] = (float)sin(a);
}
int sinusoidal(const int64_t* t, int n, int d, float* out, cudaStream_t st) {
  const int tot = n * (d / 2);
  sinusoidal_k<<<(tot + 127) / 128, 128, 0, st>>>(t, n, d, out);
  return 1;
}

// ------------------------------------------------------------------ MSE loss + gradient
template <typename T>
__global__ void mse_k(const T* __restrict__ d, const T* __restrict__ tg, size_t nvec, float scale, float inv_numel,
                      float* loss, T* __restrict__ g) {
  constexpr int V = Vec<T>::N;
  float acc = 0.f;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
    float a[V], b[V], o[V];
    ldv(d + i * V, a);
    ldv(tg + i * V, b);
#pragma unroll
    for (int k = 0; k < V; ++k) {
      const float df = a[k] - b[k];
      acc = fmaf(df, df, acc);
      o[k] = 2.0f * scale * inv_numel * df;
    }
    stv(g + i * V, o);
  }
  acc = warp_sum(acc);
  __shared__ float sh[32];
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x < 32) {
    float v = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : 0.f;
    v = warp_sum(v);
    if (threadIdx.x == 0) atomicAdd(loss, v * scale * inv_numel);
  }
}
int mse_fwd_bwd(int dt, const void* d, const void* target, size_t numel, float scale, float* loss, void* g,
                cudaStream_t st) {
  const int V = dt == DT_F32 ? 4 : 8;
  const size_t nvec = numel / V;       // numel % V == 0 is checked by the caller
  size_t blocks = (nvec + 255) / 256;
  if (blocks > 1184) blocks = 1184;
  if (blocks < 1) blocks = 1;
  const float inv = (float)(1.0 / (double)numel);
  if (dt == DT_F32)
    mse_k<float><<<(unsigned)blocks, 256, 0, st>>>((const float*)d, (const float*)target, nvec, scale, inv, loss,
                                                   (float*)g);
  else
    mse_k<bf16><<<(unsigned)blocks, 256, 0, st>>>((const bf16*)d, (const bf16*)target, nvec, scale, inv, loss,
                                                  (bf16*)g);
  return 1;
}

// ------------------------------------------------------------------ nearest 2x upsample and adjoint
template <typename T>
__global__ void upsample2_k(const T* __restrict__ in, int h, int w, int nvec, size_t total, T* __restrict__ out) {
  constexpr int V = Vec<T>::N;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    const int v = i % nvec;
    size_t p = i / nvec;                       // output pixel index n*(2h)*(2w) + Y*(2w) + X
    const int X = p % (2 * w); p /= (2 * w);
    const int Y = p % (2 * h);
    const size_t n = p / (2 * h);
    const uint4 val = *reinterpret_cast<const uint4*>(in + (((n * h + (Y >> 1)) * w + (X >> 1)) * nvec + v) * V);
    *reinterpret_cast<uint4*>(out + i * V) = val;
  }
}
template <typename T>
__global__ void upsample2_bwd_k(const T* __restrict__ gu, int h, int w, int nvec, size_t total, T* __restrict__ g) {
  constexpr int V = Vec<T>::N;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    const int v = i % nvec;
    size_t p = i / nvec;                       // low-res pixel
    const int x = p % w; p /= w;
    const int y = p % h;
    const size_t n = p / h;
    float s[V];
#pragma unroll
    for (int k = 0; k < V; ++k) s[k] = 0.f;
#pragma unroll
    for (int dy = 0; dy < 2; ++dy)
#pragma unroll
      for (int dx = 0; dx < 2; ++dx) {
        float a[V];
        ldv(gu + (((n * 2 * h + 2 * y + dy) * 2 * w + 2 * x + dx) * nvec + v) * V, a);
#pragma unroll
        for (int k = 0; k < V; ++k) s[k] += a[k];
      }
    stv(g + i * V, s);
  }
}
static unsigned ew_blocks(size_t total) {
  size_t b = (total + 255) / 256;
  if (b > 148 * 16) b = 148 * 16;
  return (unsigned)(b < 1 ? 1 : b);
}
int upsample2(int dt, const void* in, int n, int h, int w, int c, void* out, cudaStream_t st) {
  const int nvec = c / (dt == DT_F32 ? 4 : 8);
  const size_t total = (size_t)n * 4 * h * w * nvec;
  if (dt == DT_F32) upsample2_k<float><<<ew_blocks(total), 256, 0, st>>>((const float*)in, h, w, nvec, total, (float*)out);
  else upsample2_k<bf16><<<ew_blocks(total), 256, 0, st>>>((const bf16*)in, h, w, nvec, total, (bf16*)out);
  return 1;
}
int upsample2_bwd(int dt, const void* g_u, int n, int h, int w, int c, void* g_out, cudaStream_t st) {
  const int nvec = c / (dt == DT_F32 ? 4 : 8);
  const size_t total = (size_t)n * h * w * nvec;
  if (dt == DT_F32) upsample2_bwd_k<float><<<ew_blocks(total), 256, 0, st>>>((const float*)g_u, h, w, nvec, total, (float*)g_out);
  else upsample2_bwd_k<bf16><<<ew_blocks(total), 256, 0, st>>>((const bf16*)g_u, h, w, nvec, total, (bf16*)g_out);
  return 1;
}

// ------------------------------------------------------------------ dst += src
template <typename T>
__global__ void add_inplace_k(T* __restrict__ dst, const T* __restrict__ src, size_t nvec) {
  constexpr int V = Vec<T>::N;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
    float a[V], b[V];
    ldv(dst + i * V, a);
    ldv(src + i * V, b);
#pragma unroll
    for (int k = 0; k < V; ++k) a[k] += b[k];
    stv(dst + i * V, a);
  }
}
int add_inplace(int dt, void* dst, const void* src, size_t numel, cudaStream_t st) {
  const size_t nvec = numel / (dt == DT_F32 ? 4 : 8);
  if (dt == DT_F32) add_inplace_k<float><<<ew_blocks(nvec), 256, 0, st>>>((float*)dst, (const float*)src, nvec);
  else add_inplace_k<bf16><<<ew_blocks(nvec), 256, 0, st>>>((bf16*)dst, (const bf16*)src, nvec);
  return 1;
}

// ------------------------------------------------------------------ Wt[ci][k-1-r][k-1-s][co] = W[co][r][s][ci]
template <typename T>
__global__ void flip_transpose_k(const T* __restrict__ w, int cout, int kk, int cin, T* __restrict__ wt) {
  // tile transpose through shared memory: reads coalesced along ci, writes coalesced along co
  __shared__ T tile[32][33];
  const int tap = blockIdx.z;
  const int ci0 = blockIdx.x * 32, co0 = blockIdx.y * 32;
  for (int j = threadIdx.y; j < 32; j += blockDim.y) {
    const int co = co0 + j, ci = ci0 + threadIdx.x;
    if (co < cout && ci < cin) tile[j][threadIdx.x] = w[((size_t)co * kk + tap) * cin + ci];
  }
  __syncthreads();
  const int ftap = kk - 1 - tap;      // (k-1-r)*k + (k-1-s) == k*k-1 - (r*k+s)
  for (int j = threadIdx.y; j < 32; j += blockDim.y) {
    const int ci = ci0 + j, co = co0 + threadIdx.x;
    if (co < cout && ci < cin) wt[((size_t)ci * kk + ftap) * cout + co] = tile[threadIdx.x][j];
  }
}
// all conv weights of a stage in one launch per 16 tensors: blockIdx.z = entry * 9 + tap, 64 x 64 tiles.  bf16 with
// channel counts that are multiples of 8: 16-byte global accesses both ways (a tile row is 128 contiguous bytes);
// the tile is transposed on its way INTO shared memory (8 two-byte stores per 16-byte load, pitch 66 elements: a
// column walk lands on 4 different banks, 2-way conflicts) and read back as 4-byte words.
template <typename T>
__global__ void __launch_bounds__(256) flip_transpose_batch_k(const __grid_constant__ TransposeBatch b) {
  const TransposeEntry& e = b.e[blockIdx.z / 9];
  const int tap = blockIdx.z % 9, kk = e.k * e.k;
  const int ci0 = blockIdx.x * 64, co0 = blockIdx.y * 64;
  if (tap >= kk || ci0 >= e.cin || co0 >= e.cout) return;
  const int ftap = kk - 1 - tap, tx = threadIdx.x, ty = threadIdx.y, t = ty * 32 + tx;
  if (sizeof(T) == 2 && !(e.cin & 7) && !(e.cout & 7)) {
    constexpr int PITCH = 66;
    __shared__ __align__(16) uint16_t tileT[64 * PITCH];        // [ci][co]
    const uint16_t* w = (const uint16_t*)e.w;
    uint16_t* wt = (uint16_t*)e.wt;
    const int v = t & 7, r = t >> 3;            // 16-byte vector within a row, row 0..31
    uint4 in[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int co = co0 + r + 32 * h, ci = ci0 + v * 8;
      in[h] = (co < e.cout && ci < e.cin) ? *reinterpret_cast<const uint4*>(w + ((size_t)co * kk + tap) * e.cin + ci)
                                          : make_uint4(0u, 0u, 0u, 0u);
    }
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const uint32_t wd[4] = {in[h].x, in[h].y, in[h].z, in[h].w};
#pragma unroll
      for (int k = 0; k < 8; ++k)
        tileT[(v * 8 + k) * PITCH + r + 32 * h] = (uint16_t)(wd[k >> 1] >> ((k & 1) * 16));
    }
    __syncthreads();
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int cil = r + 32 * h, ci = ci0 + cil, co = co0 + v * 8;
      if (ci < e.cin && co < e.cout) {
        const uint32_t* src = reinterpret_cast<const uint32_t*>(tileT + cil * PITCH + v * 8);     // 4-byte aligned
        *reinterpret_cast<uint4*>(wt + ((size_t)ci * kk + ftap) * e.cout + co) = make_uint4(src[0], src[1], src[2], src[3]);
      }
    }
  } else {
    __shared__ T tile[64][65];
    const T* w = (const T*)e.w;
    T* wt = (T*)e.wt;
    for (int j = ty; j < 64; j += 8)
      for (int i = tx; i < 64; i += 32) {
        const int co = co0 + j, ci = ci0 + i;
        if (co < e.cout && ci < e.cin) tile[j][i] = w[((size_t)co * kk + tap) * e.cin + ci];
      }
    __syncthreads();
    for (int j = ty; j < 64; j += 8)
      for (int i = tx; i < 64; i += 32) {
        const int ci = ci0 + j, co = co0 + i;
        if (co < e.cout && ci < e.cin) wt[((size_t)ci * kk + ftap) * e.cout + co] = tile[i][j];
      }
  }
}
int flip_transpose_batch(int dt, const TransposeEntry* e, int count, cudaStream_t st) {
  int launches = 0;
  for (int i0 = 0; i0 < count; i0 += BATCH) {
    TransposeBatch b;
    b.count = count - i0 < BATCH ? count - i0 : BATCH;
    int mci = 0, mco = 0;
    for (int i = 0; i < b.count; ++i) {
      b.e[i] = e[i0 + i];
      if (b.e[i].cin > mci) mci = b.e[i].cin;
      if (b.e[i].cout > mco) mco = b.e[i].cout;
    }
    dim3 grid((mci + 63) / 64, (mco + 63) / 64, b.count * 9), block(32, 8);
    if (dt == DT_F32) flip_transpose_batch_k<float><<<grid, block, 0, st>>>(b);
    else flip_transpose_batch_k<bf16><<<grid, block, 0, st>>>(b);
    ++launches;
  }
  return launches;
}
// ------------------------------------------------------------------ pre-summed phase weights of the 4-phase upsample conv
// (kernels.h CONV_UP2).  One block = a 32 x 32 (co, ci) tile: the 9 taps are staged in shared memory as fp32, the 16
// (phase, tap) sums are formed there and written along ci (Wp) and, transposed, along co (WpT).
// The sums are formed in fp32 and rounded to the stage dtype: for bf16 that is one rounding of the WEIGHTS (2^-9 relative
// per product; measured: as much as one more bf16 store of the conv's output).  tcgen05 kind::f16 does NOT take a bf16 A
// operand with an fp16 B operand (tried: illegal instruction), so the 11 significand bits of fp16 are not available here.
template <typename T>
__global__ void __launch_bounds__(256) up2_weights_k(const T* __restrict__ w, int cout, int cin, T* __restrict__ wp,
                                                      T* __restrict__ wpt) {
  __shared__ float tile[9][32][33];
  const int ci0 = blockIdx.x * 32, co0 = blockIdx.y * 32, tx = threadIdx.x, ty = threadIdx.y;
  for (int tap = 0; tap < 9; ++tap)
    for (int j = ty; j < 32; j += 8) {
      const int co = co0 + j, ci = ci0 + tx;
      tile[tap][j][tx] = (co < cout && ci < cin) ? to_f(w[((size_t)co * 9 + tap) * cin + ci]) : 0.f;
    }
  __syncthreads();
  // R(0,0)={0}, R(0,1)={1,2}, R(1,0)={0,1}, R(1,1)={2} as [first, last] per (parity, a)
  const int lo[2][2] = {{0, 1}, {0, 2}}, hi[2][2] = {{0, 2}, {1, 2}};
  for (int q = 0; q < 16; ++q) {
    const int py = q >> 3, px = (q >> 2) & 1, a = (q >> 1) & 1, b = q & 1;      // q = (2py+px)*4 + 2a+b
    for (int j = ty; j < 32; j += 8) {
      if (wp) {           // rows co, contiguous ci
        const int co = co0 + j, ci = ci0 + tx;
        float v = 0.f;
        for (int r = lo[py][a]; r <= hi[py][a]; ++r)
          for (int s = lo[px][b]; s <= hi[px][b]; ++s) v += tile[r * 3 + s][j][tx];
        if (co < cout && ci < cin) wp[(((size_t)(q >> 2) * cout + co) * 4 + (q & 3)) * cin + ci] = from_f<T>(v);
      }
      if (wpt) {          // rows ci, contiguous co
        const int ci = ci0 + j, co = co0 + tx;
        float v = 0.f;
        for (int r = lo[py][a]; r <= hi[py][a]; ++r)
          for (int s = lo[px][b]; s <= hi[px][b]; ++s) v += tile[r * 3 + s][tx][j];
        if (co < cout && ci < cin) wpt[((size_t)ci * 16 + q) * cout + co] = from_f<T>(v);
      }
    }
  }
}
int up2_weights(int dt, const void* w, int cout, int cin, void* wp, void* wpt, cudaStream_t st) {
  dim3 grid((cin + 31) / 32, (cout + 31) / 32), block(32, 8);
  if (dt == DT_F32) up2_weights_k<float><<<grid, block, 0, st>>>((const float*)w, cout, cin, (float*)wp, (float*)wpt);
  else up2_weights_k<bf16><<<grid, block, 0, st>>>((const bf16*)w, cout, cin, (bf16*)wp, (bf16*)wpt);
  return 1;
}

int flip_transpose(int dt, const void* w, int cout, int k, int cin, void* wt, cudaStream_t st) {
  dim3 grid((cin + 31) / 32, (cout + 31) / 32, k * k), block(32, 8);
  if (dt == DT_F32) flip_transpose_k<float><<<grid, block, 0, st>>>((const float*)w, cout, k * k, cin, (float*)wt);
  else flip_transpose_k<bf16><<<grid, block, 0, st>>>((const bf16*)w, cout, k * k, cin, (bf16*)wt);
  return 1;
}

}  // namespace pulse

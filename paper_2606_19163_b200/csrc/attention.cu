// attention.cu - scaled dot-product self-attention over the pixels of a UNet level, forward and backward
// ("Each block contains Attention and ResNet layers"; formulas: oracle attn_core_*):
//   S = q k^T / sqrt(d);  P = softmax_keys(S);  o = P v
//   g_v = P^T g_o;  g_P = g_o v^T;  g_S = P (g_P - D),  D_i = sum_j P_ij g_P_ij;  g_q = g_S k / sqrt(d);  g_k = g_S^T q / sqrt(d)
// Layout: the 1x1 conv that produces q|k|v leaves them interleaved per pixel, qkv [n][T][3C] (T = H W tokens, head h owns
// channels [h d, (h+1) d) of each third), and o / g_o are [n][T][C]: no permutes, every kernel indexes the NHWC tensors.
// These are the CUDA-core kernels (fp32 arithmetic on fp32 or bf16 storage): flash-style tiles of 64 queries x 64 keys in
// shared memory, online softmax in the forward (the T x T matrix is never written), the backward recomputes P from the
// saved log-sum-exp, once per query tile (g_q) and once per key tile (g_k, g_v), so that nothing is accumulated with
// atomics (deterministic).  D is summed from P and g_P in a first sweep over the keys (not as rowsum(g_o o), which
// would read the STORED, rounded o: 2^-9 of |g_o||o| against a difference of O(1) terms).
#include "common.cuh"
#include "kernels.h"

namespace pulse {

namespace {

constexpr int BT = 64;            // tile: 64 queries x 64 keys
constexpr int PITCH = BT + 1;

struct AttnP {
  const void* qkv; const void* g_o; void* out_o; void* g_qkv;
  float* lse;                     // [2][n][heads][T]: log-sum-exp of the scaled scores | D
  int T, C, heads, d; float scale;
};

template <typename T> __device__ __forceinline__ float ld1(const T* p, size_t i) { return to_f(p[i]); }

// stage rows [r0, r0 + 64) x d channels of one third (`which`: 0 q, 1 k, 2 v) of qkv, or of a [n][T][C] tensor (stride C)
template <typename T>
__device__ __forceinline__ void load_tile(float* dst, int dp, const T* base, size_t row_stride, int r0, int Tn, int d) {
  for (int i = threadIdx.x; i < BT * d; i += blockDim.x) {
    const int r = i / d, e = i - r * d;
    dst[r * dp + e] = (r0 + r < Tn) ? ld1(base, (size_t)(r0 + r) * row_stride + e) : 0.f;
  }
}

// thread (ty, tx) of a 16 x 16 block owns rows ty + 16 i, columns tx + 16 j of a 64 x 64 tile
#define ROW(i) (ty + 16 * (i))
#define COL(j) (tx + 16 * (j))

__device__ __forceinline__ float group16_max(float v) {
#pragma unroll
  for (int o = 8; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ float group16_sum(float v) {
#pragma unroll
  for (int o = 8; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// s[i][j] = scale * sum_e A[ROW(i)][e] B[COL(j)][e]
__device__ __forceinline__ void tile_dot(const float* A, const float* Bm, int dp, int d, float scale, int ty, int tx,
                                         float (&s)[4][4]) {
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) s[i][j] = 0.f;
  for (int e = 0; e < d; ++e) {
    float a[4], b[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) a[i] = A[ROW(i) * dp + e];
#pragma unroll
    for (int j = 0; j < 4; ++j) b[j] = Bm[COL(j) * dp + e];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) s[i][j] = fmaf(a[i], b[j], s[i][j]);
  }
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) s[i][j] *= scale;
}

constexpr int MAXJ = 8;           // d <= 128

// ------------------------------------------------------------------------------ forward
template <typename T>
__global__ void __launch_bounds__(256) attn_fwd_k(const AttnP p) {
  extern __shared__ float sm[];
  const int d = p.d, dp = d + 1, Tn = p.T;
  float* Q = sm; float* K = Q + BT * dp; float* V = K + BT * dp; float* P = V + BT * dp;
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const int q0 = blockIdx.x * BT, h = blockIdx.y, n = blockIdx.z;
  const size_t rs = 3 * (size_t)p.C;
  const T* base = (const T*)p.qkv + (size_t)n * Tn * rs + (size_t)h * d;
  load_tile(Q, dp, base, rs, q0, Tn, d);
  float m[4], l[4], acc[4][MAXJ];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    m[i] = -INFINITY; l[i] = 0.f;
#pragma unroll
    for (int j = 0; j < MAXJ; ++j) acc[i][j] = 0.f;
  }
  for (int k0 = 0; k0 < Tn; k0 += BT) {
    __syncthreads();                       // previous tile fully consumed (and Q staged)
    load_tile(K, dp, base + p.C, rs, k0, Tn, d);
    load_tile(V, dp, base + 2 * p.C, rs, k0, Tn, d);
    __syncthreads();
    float s[4][4];
    tile_dot(Q, K, dp, d, p.scale, ty, tx, s);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      float mx = -INFINITY;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        if (k0 + COL(j) >= Tn) s[i][j] = -INFINITY;      // keys beyond the sequence
        mx = fmaxf(mx, s[i][j]);
      }
      mx = group16_max(mx);
      const float mn = fmaxf(m[i], mx);                  // finite: every tile holds at least one real key
      const float corr = __expf(m[i] - mn);
      float sum = 0.f;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const float e = __expf(s[i][j] - mn);
        P[ROW(i) * PITCH + COL(j)] = e;
        sum += e;
      }
      l[i] = l[i] * corr + group16_sum(sum);
      m[i] = mn;
#pragma unroll
      for (int j = 0; j < MAXJ; ++j) acc[i][j] *= corr;
    }
    __syncthreads();
    for (int c = 0; c < BT; ++c) {
      float pv[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) pv[i] = P[ROW(i) * PITCH + c];
#pragma unroll
      for (int j = 0; j < MAXJ; ++j) {
        if (COL(j) < d) {
          const float v = V[c * dp + COL(j)];
#pragma unroll
          for (int i = 0; i < 4; ++i) acc[i][j] = fmaf(pv[i], v, acc[i][j]);
        }
      }
    }
  }
  T* o = (T*)p.out_o + (size_t)n * Tn * p.C + (size_t)h * d;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int r = q0 + ROW(i);
    if (r >= Tn) continue;
    const float inv = 1.0f / l[i];
#pragma unroll
    for (int j = 0; j < MAXJ; ++j)
      if (COL(j) < d) o[(size_t)r * p.C + COL(j)] = from_f<T>(acc[i][j] * inv);
    if (tx == 0) p.lse[((size_t)n * p.heads + h) * Tn + r] = m[i] + __logf(l[i]);
  }
}

// ------------------------------------------------------------------------------ backward: g_q (one block per query tile)
template <typename T>
__global__ void __launch_bounds__(256) attn_bwd_dq_k(const AttnP p) {
  extern __shared__ float sm[];
  const int d = p.d, dp = d + 1, Tn = p.T;
  float* Q = sm; float* dO = Q + BT * dp; float* K = dO + BT * dp; float* V = K + BT * dp; float* dS = V + BT * dp;
  __shared__ float Dr[BT], Lr[BT];
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const int q0 = blockIdx.x * BT, h = blockIdx.y, n = blockIdx.z;
  const size_t rs = 3 * (size_t)p.C;
  const T* base = (const T*)p.qkv + (size_t)n * Tn * rs + (size_t)h * d;
  const T* go = (const T*)p.g_o + (size_t)n * Tn * p.C + (size_t)h * d;
  float* lse = p.lse + ((size_t)n * p.heads + h) * Tn;
  float* Dg = lse + (size_t)gridDim.z * p.heads * Tn;
  load_tile(Q, dp, base, rs, q0, Tn, d);
  load_tile(dO, dp, go, (size_t)p.C, q0, Tn, d);
  if (threadIdx.x < BT) Lr[threadIdx.x] = q0 + threadIdx.x < Tn ? lse[q0 + threadIdx.x] : 0.f;
  // first sweep over the keys: D_i = sum_j P_ij g_P_ij
  float dsum[4] = {0.f, 0.f, 0.f, 0.f};
  for (int k0 = 0; k0 < Tn; k0 += BT) {
    __syncthreads();
    load_tile(K, dp, base + p.C, rs, k0, Tn, d);
    load_tile(V, dp, base + 2 * p.C, rs, k0, Tn, d);
    __syncthreads();
    float s[4][4], gp[4][4];
    tile_dot(Q, K, dp, d, p.scale, ty, tx, s);
    tile_dot(dO, V, dp, d, 1.0f, ty, tx, gp);
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if (k0 + COL(j) < Tn) dsum[i] = fmaf(__expf(s[i][j] - Lr[ROW(i)]), gp[i][j], dsum[i]);
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    dsum[i] = group16_sum(dsum[i]);
    if (tx == 0) {
      Dr[ROW(i)] = dsum[i];
      if (q0 + ROW(i) < Tn) Dg[q0 + ROW(i)] = dsum[i];   // for the g_k / g_v kernel
    }
  }
  float acc[4][MAXJ];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < MAXJ; ++j) acc[i][j] = 0.f;
  for (int k0 = 0; k0 < Tn; k0 += BT) {
    __syncthreads();
    load_tile(K, dp, base + p.C, rs, k0, Tn, d);
    load_tile(V, dp, base + 2 * p.C, rs, k0, Tn, d);
    __syncthreads();
    float s[4][4], gp[4][4];
    tile_dot(Q, K, dp, d, p.scale, ty, tx, s);
    tile_dot(dO, V, dp, d, 1.0f, ty, tx, gp);
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const float pr = (k0 + COL(j) < Tn) ? __expf(s[i][j] - Lr[ROW(i)]) : 0.f;
        dS[ROW(i) * PITCH + COL(j)] = pr * (gp[i][j] - Dr[ROW(i)]);
      }
    __syncthreads();
    for (int c = 0; c < BT; ++c) {
      float ds[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) ds[i] = dS[ROW(i) * PITCH + c];
#pragma unroll
      for (int j = 0; j < MAXJ; ++j)
        if (COL(j) < d) {
          const float kv = K[c * dp + COL(j)];
#pragma unroll
          for (int i = 0; i < 4; ++i) acc[i][j] = fmaf(ds[i], kv, acc[i][j]);
        }
    }
  }
  T* gq = (T*)p.g_qkv + (size_t)n * Tn * rs + (size_t)h * d;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int r = q0 + ROW(i);
    if (r >= Tn) continue;
#pragma unroll
    for (int j = 0; j < MAXJ; ++j)
      if (COL(j) < d) gq[(size_t)r * rs + COL(j)] = from_f<T>(acc[i][j] * p.scale);
  }
}

// ------------------------------------------------------------------------------ backward: g_k, g_v (one block per key tile)
template <typename T>
__global__ void __launch_bounds__(256) attn_bwd_dkv_k(const AttnP p) {
  extern __shared__ float sm[];
  const int d = p.d, dp = d + 1, Tn = p.T;
  float* Q = sm; float* dO = Q + BT * dp; float* K = dO + BT * dp; float* V = K + BT * dp;
  float* Ps = V + BT * dp; float* dS = Ps + BT * PITCH;
  __shared__ float Dr[BT], Lr[BT];
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const int k0 = blockIdx.x * BT, h = blockIdx.y, n = blockIdx.z;
  const size_t rs = 3 * (size_t)p.C;
  const T* base = (const T*)p.qkv + (size_t)n * Tn * rs + (size_t)h * d;
  const T* go = (const T*)p.g_o + (size_t)n * Tn * p.C + (size_t)h * d;
  const float* lse = p.lse + ((size_t)n * p.heads + h) * Tn;
  const float* Dg = lse + (size_t)gridDim.z * p.heads * Tn;
  load_tile(K, dp, base + p.C, rs, k0, Tn, d);
  load_tile(V, dp, base + 2 * p.C, rs, k0, Tn, d);
  float gk[4][MAXJ], gv[4][MAXJ];          // rows = keys ROW(i), columns = channels COL(j)
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < MAXJ; ++j) gk[i][j] = gv[i][j] = 0.f;
  for (int q0 = 0; q0 < Tn; q0 += BT) {
    __syncthreads();
    load_tile(Q, dp, base, rs, q0, Tn, d);
    load_tile(dO, dp, go, (size_t)p.C, q0, Tn, d);
    if (threadIdx.x < BT) {
      const int r = q0 + threadIdx.x;
      Dr[threadIdx.x] = r < Tn ? Dg[r] : 0.f;
      Lr[threadIdx.x] = r < Tn ? lse[r] : 0.f;
    }
    __syncthreads();
    float s[4][4], gp[4][4];
    tile_dot(Q, K, dp, d, p.scale, ty, tx, s);           // [query ROW(i)][key COL(j)]
    tile_dot(dO, V, dp, d, 1.0f, ty, tx, gp);
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const bool in = q0 + ROW(i) < Tn && k0 + COL(j) < Tn;
        const float pr = in ? __expf(s[i][j] - Lr[ROW(i)]) : 0.f;
        Ps[ROW(i) * PITCH + COL(j)] = pr;
        dS[ROW(i) * PITCH + COL(j)] = pr * (gp[i][j] - Dr[ROW(i)]);
      }
    __syncthreads();
    for (int r = 0; r < BT; ++r) {
      float pr[4], ds[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) { pr[i] = Ps[r * PITCH + ROW(i)]; ds[i] = dS[r * PITCH + ROW(i)]; }
#pragma unroll
      for (int j = 0; j < MAXJ; ++j)
        if (COL(j) < d) {
          const float g = dO[r * dp + COL(j)], qv = Q[r * dp + COL(j)];
#pragma unroll
          for (int i = 0; i < 4; ++i) { gv[i][j] = fmaf(pr[i], g, gv[i][j]); gk[i][j] = fmaf(ds[i], qv, gk[i][j]); }
        }
    }
  }
  T* gkp = (T*)p.g_qkv + (size_t)n * Tn * rs + (size_t)h * d + p.C;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int r = k0 + ROW(i);
    if (r >= Tn) continue;
#pragma unroll
    for (int j = 0; j < MAXJ; ++j)
      if (COL(j) < d) {
        gkp[(size_t)r * rs + COL(j)] = from_f<T>(gk[i][j] * p.scale);
        gkp[(size_t)r * rs + p.C + COL(j)] = from_f<T>(gv[i][j]);
      }
  }
}
#undef ROW
#undef COL

template <typename K> void big_smem(K kernel, size_t bytes) {
  if (bytes > 48 * 1024) cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

}  // namespace

bool attn_supported(int C, int heads) { return heads > 0 && C % heads == 0 && C / heads <= 16 * MAXJ; }
size_t attn_stats_floats(int n, int heads, int T) { return (size_t)2 * n * heads * T; }

int attn_fwd(int dt, const void* qkv, int n, int T, int C, int heads, void* o, float* lse, cudaStream_t st, bool use_tc) {
  if (use_tc && attn_fwd_tc_supported(dt, C, heads)) return attn_fwd_tc(qkv, n, T, C, heads, o, lse, st);
  AttnP p{};
  p.qkv = qkv; p.out_o = o; p.lse = lse; p.T = T; p.C = C; p.heads = heads; p.d = C / heads; p.scale = 1.0f / sqrtf((float)p.d);
  dim3 grid((T + BT - 1) / BT, heads, n);
  const size_t sm = ((size_t)3 * BT * (p.d + 1) + (size_t)BT * PITCH) * sizeof(float);
  if (dt == DT_F32) { big_smem(attn_fwd_k<float>, sm); attn_fwd_k<float><<<grid, 256, sm, st>>>(p); }
  else { big_smem(attn_fwd_k<bf16>, sm); attn_fwd_k<bf16><<<grid, 256, sm, st>>>(p); }
  return 1;
}

int attn_bwd(int dt, const void* qkv, const void* g_o, int n, int T, int C, int heads, float* lse, void* g_qkv,
             cudaStream_t st, bool use_tc) {
  if (use_tc && attn_fwd_tc_supported(dt, C, heads)) return attn_bwd_tc(qkv, g_o, n, T, C, heads, lse, g_qkv, st);
  AttnP p{};
  p.qkv = qkv; p.g_o = g_o; p.g_qkv = g_qkv; p.lse = lse; p.T = T; p.C = C; p.heads = heads; p.d = C / heads;
  p.scale = 1.0f / sqrtf((float)p.d);
  dim3 grid((T + BT - 1) / BT, heads, n);
  const size_t sm1 = ((size_t)4 * BT * (p.d + 1) + (size_t)BT * PITCH) * sizeof(float);
  const size_t sm2 = ((size_t)4 * BT * (p.d + 1) + (size_t)2 * BT * PITCH) * sizeof(float);
  if (dt == DT_F32) {
    big_smem(attn_bwd_dq_k<float>, sm1); big_smem(attn_bwd_dkv_k<float>, sm2);
    attn_bwd_dq_k<float><<<grid, 256, sm1, st>>>(p);
    attn_bwd_dkv_k<float><<<grid, 256, sm2, st>>>(p);
  } else {
    big_smem(attn_bwd_dq_k<bf16>, sm1); big_smem(attn_bwd_dkv_k<bf16>, sm2);
    attn_bwd_dq_k<bf16><<<grid, 256, sm1, st>>>(p);
    attn_bwd_dkv_k<bf16><<<grid, 256, sm2, st>>>(p);
  }
  return 2;
}

}  // namespace pulse

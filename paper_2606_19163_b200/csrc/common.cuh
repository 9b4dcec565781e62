// common.cuh - element types, 16-byte vector access, small device helpers.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdlib>
#include <utility>

#include "toggles.h"

namespace pulse {

typedef __nv_bfloat16 bf16;

// ---- programmatic dependent launch (PDL) ------------------------------------------------------------------
// Kernels launched through launch_pdl may start while the previous kernel of the stream is still draining: their
// CTAs are scheduled as SMs free up and run their prologue (barrier init, TMEM allocation, tensor-map prefetch),
// then block in pdl_wait() until the previous grid has completed and its writes are visible.  Every such kernel
// calls pdl_wait() before its first global-memory access and pdl_launch_dependents() right after it.
// PULSE_NO_PDL=1 launches them as ordinary stream-ordered kernels (both calls are then no-ops).
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
inline bool pdl_enabled() { return !toggles().no_pdl; }
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                              Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = pdl_enabled() ? 1 : 0;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

template <typename T> struct Vec;                 // 16-byte vector of T
template <> struct Vec<float> { static constexpr int N = 4; };
template <> struct Vec<bf16>  { static constexpr int N = 8; };

__device__ __forceinline__ float to_f(float v) { return v; }
__device__ __forceinline__ float to_f(bf16 v) { return __bfloat162float(v); }
template <typename T> __device__ __forceinline__ T from_f(float v);
template <> __device__ __forceinline__ float from_f<float>(float v) { return v; }
template <> __device__ __forceinline__ bf16 from_f<bf16>(float v) { return __float2bfloat16_rn(v); }

// 16 raw bytes -> 4 floats (fp32 tensor) or 8 floats (bf16 tensor)
__device__ __forceinline__ void unpack(const uint4& v, float (&o)[4]) {
  o[0] = __uint_as_float(v.x); o[1] = __uint_as_float(v.y); o[2] = __uint_as_float(v.z); o[3] = __uint_as_float(v.w);
}
__device__ __forceinline__ void unpack(const uint4& v, float (&o)[8]) {
  const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    o[2 * i] = __uint_as_float(w[i] << 16);
    o[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
  }
}
// load Vec<T>::N consecutive elements (16-byte aligned) into floats
__device__ __forceinline__ void ldv(const float* p, float (&o)[4]) { unpack(*reinterpret_cast<const uint4*>(p), o); }
__device__ __forceinline__ void ldv(const bf16* p, float (&o)[8]) { unpack(*reinterpret_cast<const uint4*>(p), o); }
__device__ __forceinline__ void stv(float* p, const float (&o)[4]) {
  *reinterpret_cast<float4*>(p) = make_float4(o[0], o[1], o[2], o[3]);
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&h);
}
__device__ __forceinline__ void stv(bf16* p, const float (&o)[8]) {
  uint4 v;
  v.x = pack_bf16(o[0], o[1]); v.y = pack_bf16(o[2], o[3]);
  v.z = pack_bf16(o[4], o[5]); v.w = pack_bf16(o[6], o[7]);
  *reinterpret_cast<uint4*>(p) = v;
}

// ---- packed fp32 pairs (sm_100 FFMA2 / FMUL2 / FADD2: one issue slot for two lanes of arithmetic).
// A pair is (lo, hi) = two neighbouring channels.
typedef unsigned long long f2_t;
__device__ __forceinline__ f2_t pk2(float lo, float hi) { f2_t r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void upk2(f2_t v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f2_t fma2(f2_t a, f2_t b, f2_t c) { f2_t r; asm("fma.rn.ftz.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ f2_t mul2(f2_t a, f2_t b) { f2_t r; asm("mul.rn.ftz.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f2_t add2(f2_t a, f2_t b) { f2_t r; asm("add.rn.ftz.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
// two bf16 of one 32-bit word -> fp32 pair (element 2j in the low half)
__device__ __forceinline__ f2_t bf2(uint32_t w) { return pk2(__uint_as_float(w << 16), __uint_as_float(w & 0xffff0000u)); }

__device__ __forceinline__ float sigmoidf_(float y) { return 1.0f / (1.0f + __expf(-y)); }
__device__ __forceinline__ float siluf_(float y) { return y * sigmoidf_(y); }
__device__ __forceinline__ float silu_gradf_(float y) {
  float s = sigmoidf_(y);
  return s * (1.0f + y * (1.0f - s));
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

}  // namespace pulse

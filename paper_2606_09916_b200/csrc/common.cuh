// common.cuh -- shared device helpers of libikv (sm_100a). Not shared with oracle/.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

namespace ikv {

typedef __nv_bfloat16 bf16;

constexpr int CLS_DEAD = 0, CLS_FORCED = 1, CLS_CAND = 2;

// 16-byte streaming load that does not allocate in L1 (keys/values are read once per pass)
__device__ __forceinline__ uint4 ld_stream16(const void* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}

__device__ __forceinline__ float bf16lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16hi(uint32_t u) { return __uint_as_float(u & 0xffff0000u); }

// Elem<T>: VEC elements of T per 16-byte load, converted exactly to fp32
template <typename T>
struct Elem;
template <>
struct Elem<float> {
  static constexpr int VEC = 4;
  __device__ __forceinline__ static void unpack(const uint4& t, float (&v)[4]) {
    v[0] = __uint_as_float(t.x); v[1] = __uint_as_float(t.y);
    v[2] = __uint_as_float(t.z); v[3] = __uint_as_float(t.w);
  }
};
template <>
struct Elem<bf16> {
  static constexpr int VEC = 8;
  __device__ __forceinline__ static void unpack(const uint4& t, float (&v)[8]) {
    v[0] = bf16lo(t.x); v[1] = bf16hi(t.x); v[2] = bf16lo(t.y); v[3] = bf16hi(t.y);
    v[4] = bf16lo(t.z); v[5] = bf16hi(t.z); v[6] = bf16lo(t.w); v[7] = bf16hi(t.w);
  }
};

__device__ __forceinline__ int classify(int32_t slot, int j, int32_t dead, int pi, int qs, int qe) {
  if (slot == dead) return CLS_DEAD;
  if (j < pi || (j >= qs && j < qe)) return CLS_FORCED;
  return CLS_CAND;
}

__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ int warp_sum_i(int v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Exclusive block scan of one int per thread for blockDim.x == 1024 (32 warps).
// `warp_tot` is a 32-int shared array.  Returns the exclusive prefix; *total = block sum.
__device__ __forceinline__ int block_excl_scan_1024(int v, int* warp_tot, int* total) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int n = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += n;
  }
  __syncthreads();  // protect warp_tot reuse
  if (lane == 31) warp_tot[wid] = inc;
  __syncthreads();
  int wv = warp_tot[lane];
  int winc = wv;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int n = __shfl_up_sync(0xffffffffu, winc, o);
    if (lane >= o) winc += n;
  }
  const int wbase = __shfl_sync(0xffffffffu, winc - wv, wid);
  *total = __shfl_sync(0xffffffffu, winc, 31);
  return wbase + inc - v;
}

}  // namespace ikv

// Shared definitions of the KVarN CUDA library (sm_100a): record layout,
// storage-format conversions, small warp helpers.  See include/kvarn.h for the
// boundary and DESIGN.md for the data layout in HBM.
#pragma once

#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_fp8.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/kvarn.h"

namespace kvarn {

constexpr int D = KVARN_HEAD_DIM;   // channels per head
constexpr int G = KVARN_CHUNK;      // tokens per chunk
constexpr int AUX_BYTES = 512;      // 128 fp8 s1 + 128 fp8 s2 + 128 fp16 z

__host__ __device__ constexpr int codes_bytes(int bits) { return D * G * bits / 8; }
__host__ __device__ constexpr int record_bytes(int bits) { return codes_bytes(bits) + AUX_BYTES; }
__host__ __device__ constexpr int row_bytes(int bits) { return D * bits / 8; }  // one code row
__host__ __device__ constexpr int s1_off(int bits) { return codes_bytes(bits); }
__host__ __device__ constexpr int s2_off(int bits) { return codes_bytes(bits) + 128; }
__host__ __device__ constexpr int z_off(int bits) { return codes_bytes(bits) + 256; }

// Code rows are stored "segment-major": the 16-byte segment s of row r (a row =
// the 128 codes of one token (K) / one channel (V), little-endian, element e at
// bit bits*(e % (8/bits)) of byte e*bits/8) sits at  s*2048 + r*16, so that 128
// threads reading one segment of their own row touch consecutive 16-byte words.
__host__ __device__ constexpr int code_off(int row, int byte_in_row) {
  return (byte_in_row >> 4) * 2048 + row * 16 + (byte_in_row & 15);
}
// "K position" of element e of a code row inside the tensor-core A operand:
// the decode kernel expands a packed 32-bit word W with  W & (mask << bits*j), so
// byte b of A column (8/bits)*w + j holds element (32/bits)*w + (8/bits)*b + j.
// kpos = 4*column + b.
__host__ __device__ constexpr int kpos_of_elem(int bits, int e) {
  return bits == 2 ? ((e & ~15) | ((e & 3) << 2) | ((e >> 2) & 3)) : ((e & ~7) | ((e & 1) << 2) | ((e >> 1) & 3));
}
__host__ __device__ constexpr int elem_of_kpos(int bits, int k) {
  return bits == 2 ? ((k & ~15) | ((k & 3) << 2) | ((k >> 2) & 3)) : ((k & ~7) | ((k & 3) << 1) | ((k >> 2) & 1));
}
// The per-channel aux arrays of K records (s1, z) are stored so that lane l of
// the decode kernel's B-operand builder, which owns K positions l, l+32, l+64,
// l+96, reads its four values contiguously: index 4*(kpos & 31) + (kpos >> 5).
__host__ __device__ constexpr int kaux_of_elem(int bits, int e) {
  return 4 * (kpos_of_elem(bits, e) & 31) + (kpos_of_elem(bits, e) >> 5);
}

// ---- storage formats -------------------------------------------------------
// FP8 E4M3 (finite, max 448), round-to-nearest-even, saturating (DESIGN R9).
__host__ __device__ inline uint8_t f32_to_e4m3(float x) {
  return (uint8_t)__nv_cvt_float_to_fp8(x, __NV_SATFINITE, __NV_E4M3);
}
__host__ __device__ inline float e4m3_to_f32(uint8_t b) {
  __half_raw h = __nv_cvt_fp8_to_halfraw((__nv_fp8_storage_t)b, __NV_E4M3);
  return __half2float(__half(h));
}
__host__ __device__ inline uint16_t f32_to_f16_bits(float x) {
  __half h = __float2half_rn(x);
  return __half_as_ushort(h);
}
__host__ __device__ inline float f16_bits_to_f32(uint16_t b) {
  return __half2float(__ushort_as_half(b));
}

#ifdef __CUDACC__
__device__ __forceinline__ float bf16_bits_to_f32(uint32_t b16) { return __uint_as_float(b16 << 16); }

// two packed e4m3 bytes (low 16 bits of v) -> two floats
__device__ __forceinline__ float2 e4m3x2_to_f32x2(uint16_t v) {
  uint32_t h2;
  asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h2) : "h"(v));
  __half2 h = *reinterpret_cast<__half2*>(&h2);
  return __half22float2(h);
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int m = 16; m > 0; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
  return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int m = 16; m > 0; m >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, m));
  return v;
}

// In-register Walsh-Hadamard butterflies over 128 values spread as 4 per lane
// (element index e = 4*lane + j): used for the single-vector transforms of
// decode (q and the output).  Unnormalised.
__device__ __forceinline__ void fwht128_lane4(float (&v)[4], int lane) {
  // bits 0,1: inside the lane
  float a0 = v[0] + v[1], a1 = v[0] - v[1], a2 = v[2] + v[3], a3 = v[2] - v[3];
  v[0] = a0 + a2; v[1] = a1 + a3; v[2] = a0 - a2; v[3] = a1 - a3;
  // bits 2..6: across lanes (lane bit m <-> element bit 4m)
#pragma unroll
  for (int m = 1; m < 32; m <<= 1) {
    const float sgn = (lane & m) ? -1.f : 1.f;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      float p = __shfl_xor_sync(0xffffffffu, v[j], m);
      v[j] = fmaf(sgn, v[j], p);
    }
  }
}
#endif  // __CUDACC__

}  // namespace kvarn

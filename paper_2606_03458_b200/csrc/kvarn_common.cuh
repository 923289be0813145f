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

// ---- record layout ---------------------------------
// The decode kernel contracts with warp-level IMMA m16n8k32 (u8 x s8/u8 -> s32):
// the 128 code rows of a record (K: one row per token, V: one row per channel;
// a row = 128 codes, little-endian, element e at bit bits*(e % (8/bits)) of byte
// e*bits/8) are the M rows.  "Slot" s = 32*warp + 16*mtile + 8*rho + g names the
// MMA row that thread (g = lane>>2, t = lane&3) of `warp` holds in A registers
// a[rho] / a[rho+2] of m-tile `mtile`.  A packed 32-bit word W of a row expands
// with one LOP3 per register,  W & (mask << bits*j),  into the four k-bytes of
// one A register, so thread t needs words t, t+4 (, t+8, t+12 at 4-bit) of its
// four rows; they are stored so that each (warp, mtile[, rho]) is one conflict-
// free LDS.128 per lane.
__host__ __device__ constexpr int code_off(int bits, int slot, int byte_in_row) {
  const int wi = byte_in_row >> 2, bb = byte_in_row & 3;
  const int w = slot >> 5, mt = (slot >> 4) & 1, rho = (slot >> 3) & 1, g = slot & 7;
  const int t = wi & 3, q = wi >> 2;
  return bits == 2 ? w * 1024 + mt * 512 + (4 * g + t) * 16 + rho * 8 + q * 4 + bb
                   : w * 2048 + mt * 1024 + rho * 512 + (4 * g + t) * 16 + q * 4 + bb;
}
// Position of element e of a code row in the contraction (K) dimension: k-step
// kappa (32 positions each) and position p inside it.  All codes of one k-step
// sit at the same bit offset bits*j inside their byte (2-bit: j = kappa, 4-bit:
// j = kappa & 1); the B operand compensates with a power of two.
__host__ __device__ constexpr int kstep_of_elem(int bits, int e) {
  return bits == 2 ? (e & 3) : (2 * (e >> 6) + (e & 1));
}
__host__ __device__ constexpr int kpos_of_elem(int bits, int e) {   // p = 16*half + 4*t' + b
  return bits == 2 ? (16 * (e >> 6) + 4 * ((e >> 4) & 3) + ((e >> 2) & 3))
                   : (16 * ((e >> 5) & 1) + 4 * ((e >> 3) & 3) + ((e >> 1) & 3));
}
// B-operand builder lane that owns element e:  lane = 8*kappa + 4*half + t',  its b-th value.
__host__ __device__ constexpr int kaux_of_elem(int bits, int e) {
  return 4 * (8 * kstep_of_elem(bits, e) + (kpos_of_elem(bits, e) >> 2)) + (kpos_of_elem(bits, e) & 3);
}
// K records: MMA row slot of token tau.  Chosen so that the four tokens a thread
// sees in its C fragments (mtile, rho) are the four k-bytes b = 2*mtile + rho of
// one B-operand word of the value contraction (k-step = warp, half = g>>2, t' = g&3).
__host__ __device__ constexpr int slot_of_token(int bits, int tau) {
  return bits == 2
             ? 32 * (tau & 3) + 16 * ((tau >> 3) & 1) + 8 * ((tau >> 2) & 1) + ((((tau >> 6) & 1) << 2) | ((tau >> 4) & 3))
             : 32 * ((((tau >> 6) & 1) << 1) | (tau & 1)) + 16 * ((tau >> 2) & 1) + 8 * ((tau >> 1) & 1) +
                   ((((tau >> 5) & 1) << 2) | ((tau >> 3) & 3));
}
// Aux arrays: per-token arrays (K.s2, V.s1, V.z) are stored at index slot_of_token(tau);
// K.s1 and K.z (per channel) at index kaux_of_elem(c); V.s2 (per channel) at index c.

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

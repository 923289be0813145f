// Hadamard arrangement around the attention layer (App. A, Fig. 7):
//   - the two ONLINE head-wise transforms "after the RoPE-embedding" of q and K, fused with the rotary
//     embedding itself (rope_hadamard_kernel), so that a cache written with rotate_k = 0 and read with
//     rotate_k = 0 sees already-rotated K and q;
//   - the two ABSORBED transforms merged offline into W_V and W_O (hadamard_rows_kernel over the 128-wide
//     column groups of W_V, hadamard_row_groups_kernel over the 128-row groups of W_O), after which V is
//     produced rotated (rotate_v = 0) and the rotated attention output is consumed by W_O' unchanged.
// All three are streaming kernels: one read and one write of every element, bound by HBM.
#pragma once

#include "kvarn_common.cuh"

namespace kvarn {

constexpr float HAD_NORM = 0.08838834764831845f;   // 1 / sqrt(128)

template <typename T> __device__ __forceinline__ void ld4(const T* p, float (&v)[4]);
template <> __device__ __forceinline__ void ld4<float>(const float* p, float (&v)[4]) {
  const float4 a = *reinterpret_cast<const float4*>(p);
  v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w;
}
template <> __device__ __forceinline__ void ld4<__nv_bfloat16>(const __nv_bfloat16* p, float (&v)[4]) {
  const uint2 u = *reinterpret_cast<const uint2*>(p);
  v[0] = __uint_as_float(u.x << 16); v[1] = __uint_as_float(u.x & 0xffff0000u);
  v[2] = __uint_as_float(u.y << 16); v[3] = __uint_as_float(u.y & 0xffff0000u);
}
template <typename T> __device__ __forceinline__ void st4(T* p, const float (&v)[4]);
template <> __device__ __forceinline__ void st4<float>(float* p, const float (&v)[4]) {
  *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
}
template <> __device__ __forceinline__ void st4<__nv_bfloat16>(__nv_bfloat16* p, const float (&v)[4]) {
  const __nv_bfloat162 a = __floats2bfloat162_rn(v[0], v[1]), b = __floats2bfloat162_rn(v[2], v[3]);
  uint2 u;
  u.x = *reinterpret_cast<const uint32_t*>(&a); u.y = *reinterpret_cast<const uint32_t*>(&b);
  *reinterpret_cast<uint2*>(p) = u;
}

// One warp per 128-element group (a head's slice of one row): y = RoPE(x) H / sqrt(128).
// cos / sin: [n_tok][64] fp32 (half-split convention: channel c < 64 pairs with c + 64), or null = no RoPE.
// rotate = 0 leaves out the Hadamard (plain RoPE).  Group index = tok * n_heads + head.
constexpr int ROT_GPW = 4;   // groups per warp: all loads of a warp's groups are issued before the first butterfly
template <typename T>
__global__ void __launch_bounds__(256) rope_hadamard_kernel(const T* __restrict__ x, const float* __restrict__ cs,
                                                            const float* __restrict__ sn, T* __restrict__ y,
                                                            long long n_groups, int n_heads, int rotate) {
  const int lane = threadIdx.x & 31;
  const long long g0 = ((long long)blockIdx.x * 8 + (threadIdx.x >> 5)) * ROT_GPW;
  if (g0 >= n_groups) return;
  const int c = 4 * (lane & 15);
  float v[ROT_GPW][4], cc[ROT_GPW][4], ss[ROT_GPW][4];
#pragma unroll
  for (int u = 0; u < ROT_GPW; ++u) {
    const long long grp = g0 + u;
    if (grp < n_groups) {
      ld4<T>(x + grp * D + 4 * lane, v[u]);
      if (cs) {
        const long long tok = grp / n_heads;
        ld4<float>(cs + tok * 64 + c, cc[u]);
        ld4<float>(sn + tok * 64 + c, ss[u]);
      }
    }
  }
  const float sg = lane < 16 ? -1.f : 1.f;   // y[c] = x[c] cos - x[c+64] sin;  y[c+64] = x[c+64] cos + x[c] sin
#pragma unroll
  for (int u = 0; u < ROT_GPW; ++u) {
    const long long grp = g0 + u;
    if (grp >= n_groups) break;   // warp-uniform
    if (cs) {
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const float other = __shfl_xor_sync(0xffffffffu, v[u][j], 16);
        v[u][j] = fmaf(v[u][j], cc[u][j], sg * other * ss[u][j]);
      }
    }
    if (rotate) {
      fwht128_lane4(v[u], lane);
#pragma unroll
      for (int j = 0; j < 4; ++j) v[u][j] *= HAD_NORM;
    }
    st4<T>(y + grp * D + 4 * lane, v[u]);
  }
}

// W' = blockdiag(H / sqrt(128)) W for a row-major [n_rows][n_cols] matrix, n_rows a multiple of 128: every group
// of 128 consecutive ROWS is transformed down the columns (W_O of P:332).  CTA = 128 rows x 32 columns, staged
// through shared memory so that global accesses stay coalesced along the columns.
template <typename T>
__global__ void __launch_bounds__(128) hadamard_row_groups_kernel(const T* __restrict__ w, T* __restrict__ out,
                                                                  long long n_cols) {
  __shared__ float tile[32][129];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const long long r0 = (long long)blockIdx.y * 128, c0 = (long long)blockIdx.x * 32;
  const bool col_ok = c0 + lane < n_cols;
#pragma unroll 4
  for (int r = warp; r < 128; r += 4) {
    float f = 0.f;
    if (col_ok) {
      if constexpr (sizeof(T) == 4) f = w[(r0 + r) * n_cols + c0 + lane];
      else f = __bfloat162float(w[(r0 + r) * n_cols + c0 + lane]);
    }
    tile[lane][r] = f;
  }
  __syncthreads();
  for (int c = warp; c < 32; c += 4) {
    float v[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) v[j] = tile[c][4 * lane + j];
    fwht128_lane4(v, lane);
#pragma unroll
    for (int j = 0; j < 4; ++j) tile[c][4 * lane + j] = v[j] * HAD_NORM;
  }
  __syncthreads();
  if (col_ok) {
#pragma unroll 4
    for (int r = warp; r < 128; r += 4) {
      const float f = tile[lane][r];
      if constexpr (sizeof(T) == 4) out[(r0 + r) * n_cols + c0 + lane] = f;
      else out[(r0 + r) * n_cols + c0 + lane] = __float2bfloat16_rn(f);
    }
  }
}

}  // namespace kvarn

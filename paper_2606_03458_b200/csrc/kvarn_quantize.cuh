// KVarN write path: one CTA = one (128 channel x 128 token) tile, held entirely
// in registers.  Hadamard -> Algorithm 1 VarN -> RTN
// (Eq. 1) -> FP8/FP8/FP16 aux + packed codes.
//
// Thread layout (256 threads = 8 warps): warp w owns tokens 16w..16w+15; within
// the warp lj = lane>>4 picks 8 of them (t0 = 16w + 8lj) and li = lane&15 picks
// 8 channels (c0 = 8li).  A thread holds T[c0+k][t0+i] for i,k in 0..7 as
// float2 pairs along the channel index, so every inner loop is packed f32x2
// arithmetic (FFMA2 is the full-rate fp32 instruction on sm_100).
//
// Algorithm 1 needs, per iteration, the variance of every column (token) and of
// every row (channel) of C = T / S_c / S_r.  Since the scales are constant along
// the reduced axis they factor out:
//   Var_c(C[:,t]) = b_t^2 * Var_c(a_c T[c,t]),   Var_t(C[c,:]) = a_c^2 * Var_t(b_t T[c,t])
// with a = 1/S_r, b = 1/S_c, so a half-step is one pass of (mul, add, fma) over
// the register tile plus a reduction: in-warp for tokens (transpose-reduce over
// the 16 lanes sharing a token), through shared memory for channels.  Row
// variances after a row update follow analytically (the row was rescaled by a
// constant), and the column variances needed by Imb(C_k) are exactly the ones
// the next iteration's first half-step computes -- so K iterations cost K+1
// column passes and K+1 row passes.
#pragma once

#include <type_traits>

#include "kvarn_common.cuh"

namespace kvarn {

struct VarnConsts {
  int iters;
  float var_min, var_max, log_lo, log_hi;
  int aux_round;   // 1: RTN against the stored FP8 / FP16 parameters (kvarn_params::aux_round)
};

struct QuantDebug {
  int32_t* k_best;  // [tile] for this kind, or null
  float* imb;       // [tile][KVARN_MAX_ITERS+1]
  float* aux;       // [tile][3][128]
};

template <int BITS>
struct QuantSmem {
  alignas(16) float part[8][2][128];  // cross-warp partials (row sums / min-max)
  float a[128];           // 1 / S_r  (per channel)
  alignas(16) float b[128];    // 1 / S_c  (per token)
  alignas(16) float mu[128];   // mean over the tile's tokens of T[c, :] (the channel offsets of P:127): pivot of the row passes
  float bbar;             // mean over tokens of b (one column update old, see row_partials)
  // per iterate k = 0..iters: column / row variances of C_k and the log-scales that produced it;
  // the best iterate (Alg. 1 lines 7, 18) is selected once, after the loop
  alignas(16) float cvh[KVARN_MAX_ITERS + 1][128];
  alignas(16) float rvh[KVARN_MAX_ITERS + 1][128];
  float Lch[KVARN_MAX_ITERS + 1][128];
  float Lrh[KVARN_MAX_ITERS + 1][128];
  float imb[KVARN_MAX_ITERS + 1];
  alignas(16) float Sc[128];   // best scales
  alignas(16) float Sr[128];
  alignas(16) float inv_s[128];
  alignas(16) float z[128];
  alignas(16) uint8_t rec[record_bytes(BITS)];
};

__device__ __forceinline__ float2 f2(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __ffma2_rn(b, f2(-1.f, -1.f), a); }

// 16 values per lane, 16 lanes (xor masks 8,4,2,1) -> 1 value per lane, summed
// over the 16 lanes.  Lane li ends with value index  ((li>>3)&1)*8 + (li&7).
template <class Op>
__device__ __forceinline__ float xreduce16(float (&v)[16], int li, Op op) {
  {
    const bool up = li & 8;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      float send = up ? v[j] : v[j + 8], keep = up ? v[j + 8] : v[j];
      v[j] = op(keep, __shfl_xor_sync(0xffffffffu, send, 8));
    }
  }
  {
    const bool up = li & 4;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      float send = up ? v[j] : v[j + 4], keep = up ? v[j + 4] : v[j];
      v[j] = op(keep, __shfl_xor_sync(0xffffffffu, send, 4));
    }
  }
  {
    const bool up = li & 2;
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      float send = up ? v[j] : v[j + 2], keep = up ? v[j + 2] : v[j];
      v[j] = op(keep, __shfl_xor_sync(0xffffffffu, send, 2));
    }
  }
  {
    const bool up = li & 1;
    float send = up ? v[0] : v[1], keep = up ? v[1] : v[0];
    v[0] = op(keep, __shfl_xor_sync(0xffffffffu, send, 1));
  }
  return v[0];
}

// MUFU forms for the inner loop of Alg. 1 (relative error ~2^-22 per call, an order below the
// 1e-5 tolerance on the scales after 2 x 8 half-steps; the stored scales use expf once at the end)
__device__ __forceinline__ float fast_log2(float x) { float y; asm("lg2.approx.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float fast_exp2(float x) { float y; asm("ex2.approx.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

constexpr float RTN_MAGIC = 12582912.0f;   // 1.5 * 2^23: (t + MAGIC) - MAGIC = rint(t), ties to even, for |t| < 2^22

struct OpAdd { __device__ float operator()(float a, float b) const { return a + b; } };
struct OpMin { __device__ float operator()(float a, float b) const { return fminf(a, b); } };

// Quantise the register tile x (x[i][kp] = channels c0+2kp,+1 of token t0+i, RAW
// un-rotated values) and write the record to rec_out (global, 16-B aligned).
// Must be called by all 256 threads of the CTA.
template <int BITS>
__device__ void quantize_tile(float2 (&x)[8][4], const int kind, const bool rotate,
                              const VarnConsts vc, uint8_t* __restrict__ rec_out,
                              const QuantDebug dbg, const long long tile_idx,
                              QuantSmem<BITS>& sm) {
  constexpr int LV = (1 << BITS) - 1;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int li = lane & 15, lj = lane >> 4;
  const int c0 = 8 * li, t0 = 16 * warp + 8 * lj;
  const int tok_own = t0 + (li & 7);  // token whose column statistics this lane finalises
  const float inv_n = 1.f / 128.f;

  // ---- Q1: Hadamard along channels, Y = X H / sqrt(128) -----------------------
  if (rotate) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
#pragma unroll
      for (int kp = 0; kp < 4; ++kp) x[i][kp] = f2(x[i][kp].x + x[i][kp].y, x[i][kp].x - x[i][kp].y);
      float2 n0 = add2(x[i][0], x[i][1]), n1 = sub2(x[i][0], x[i][1]);
      float2 n2 = add2(x[i][2], x[i][3]), n3 = sub2(x[i][2], x[i][3]);
      x[i][0] = add2(n0, n2); x[i][1] = add2(n1, n3);
      x[i][2] = sub2(n0, n2); x[i][3] = sub2(n1, n3);
    }
#pragma unroll
    for (int m = 1; m < 16; m <<= 1) {
      const float s = (li & m) ? -1.f : 1.f;
      const float2 sg = f2(s, s);
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int kp = 0; kp < 4; ++kp) {
          float2 p = f2(__shfl_xor_sync(0xffffffffu, x[i][kp].x, m),
                        __shfl_xor_sync(0xffffffffu, x[i][kp].y, m));
          x[i][kp] = fma2(sg, x[i][kp], p);
        }
    }
    const float2 r = f2(0.08838834764831845f, 0.08838834764831845f);
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
      for (int kp = 0; kp < 4; ++kp) x[i][kp] = mul2(x[i][kp], r);
  }

  // ---- Q2: Algorithm 1 ----------------------------------------------------------
  float2 a2[4];  // 1/S_r of own channels
  float b[8];    // 1/S_c of own tokens
#pragma unroll
  for (int kp = 0; kp < 4; ++kp) a2[kp] = f2(1.f, 1.f);
#pragma unroll
  for (int i = 0; i < 8; ++i) b[i] = 1.f;

  float Lc = 0.f, b_own = 1.f;  // log column scale of tok_own
  float Lr = 0.f, a_own = 1.f;  // log row scale of channel tid (tid < 128)

  // row half-step, part 1: per-channel sums of u and u^2 over this warp's 16 tokens -> sm.part[warp][stat][channel],
  // with u = b_t T[c,t] (PIV = false) or u = b_t T[c,t] - mu_c bbar (PIV = true).  The variance does not depend on the
  // pivot; the single-pass form E[u^2] - E[u]^2 does, in fp32: channels whose offset is tens to hundreds of standard
  // deviations ("in some cases have large offsets") would lose 3 .. 6 digits without it.  mu_c bbar is the row
  // mean of b_t T up to the correlation of b with the centred data, so E[u] stays at the size of the standard
  // deviation.  A tile takes the pivoted form only if pass 0 finds a channel with |mean| > 4 std (CTA-uniform flag).
  auto row_partials = [&](auto piv_tag, const float bbar) {
    constexpr bool PIV = decltype(piv_tag)::value;
    float2 s1[4], s2[4], npiv[4];
    if constexpr (PIV) {
      const float4* pm = reinterpret_cast<const float4*>(&sm.mu[c0]);
      const float4 m0 = pm[0], m1 = pm[1];
      const float2 nb = f2(-bbar, -bbar);
      npiv[0] = mul2(f2(m0.x, m0.y), nb); npiv[1] = mul2(f2(m0.z, m0.w), nb);
      npiv[2] = mul2(f2(m1.x, m1.y), nb); npiv[3] = mul2(f2(m1.z, m1.w), nb);
    }
#pragma unroll
    for (int kp = 0; kp < 4; ++kp) { s1[kp] = f2(0.f, 0.f); s2[kp] = f2(0.f, 0.f); }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const float2 bb = f2(b[i], b[i]);
#pragma unroll
      for (int kp = 0; kp < 4; ++kp) {
        float2 u = PIV ? fma2(x[i][kp], bb, npiv[kp]) : mul2(x[i][kp], bb);
        s1[kp] = add2(s1[kp], u);
        s2[kp] = fma2(u, u, s2[kp]);
      }
    }
    // combine the two token halves (lanes l, l^16): lj=0 keeps the sums, lj=1 the squares
    float4 o0, o1;
    {
      float send[8], keep[8];
#pragma unroll
      for (int kp = 0; kp < 4; ++kp) {
        send[2 * kp] = lj ? s1[kp].x : s2[kp].x; send[2 * kp + 1] = lj ? s1[kp].y : s2[kp].y;
        keep[2 * kp] = lj ? s2[kp].x : s1[kp].x; keep[2 * kp + 1] = lj ? s2[kp].y : s1[kp].y;
      }
#pragma unroll
      for (int j = 0; j < 8; ++j) keep[j] += __shfl_xor_sync(0xffffffffu, send[j], 16);
      o0 = make_float4(keep[0], keep[1], keep[2], keep[3]);
      o1 = make_float4(keep[4], keep[5], keep[6], keep[7]);
    }
    float4* dst = reinterpret_cast<float4*>(&sm.part[warp][lj][c0]);
    dst[0] = o0; dst[1] = o1;
  };

  // row half-step, part 2 (threads 0..127, channel = tid): raw row variance of
  // the current C.
  auto row_variance_own = [&]() -> float {
    float s1 = 0.f, s2 = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) { s1 += sm.part[w][0][tid]; s2 += sm.part[w][1][tid]; }
    const float mean = s1 * inv_n;
    return fmaxf(fmaf(-mean, mean, s2 * inv_n), 0.f) * (a_own * a_own);
  };

  auto reload_a = [&]() {
    const float4* src = reinterpret_cast<const float4*>(&sm.a[c0]);
    float4 v0 = src[0], v1 = src[1];
    a2[0] = f2(v0.x, v0.y); a2[1] = f2(v0.z, v0.w); a2[2] = f2(v1.x, v1.y); a2[3] = f2(v1.z, v1.w);
  };
  auto reload_b = [&]() {
    const float4* src = reinterpret_cast<const float4*>(&sm.b[t0]);
    float4 v0 = src[0], v1 = src[1];
    b[0] = v0.x; b[1] = v0.y; b[2] = v0.z; b[3] = v0.w; b[4] = v1.x; b[5] = v1.y; b[6] = v1.z; b[7] = v1.w;
  };

  // Imb(C) (DESIGN R1) from the 128 column and 128 row variances in shared memory
  auto imbalance = [&](int k) -> float {
    const float4 c4 = reinterpret_cast<const float4*>(sm.cvh[k])[lane];
    const float4 r4 = reinterpret_cast<const float4*>(sm.rvh[k])[lane];
    float mx = fmaxf(fmaxf(fmaxf(c4.x, c4.y), fmaxf(c4.z, c4.w)), fmaxf(fmaxf(r4.x, r4.y), fmaxf(r4.z, r4.w)));
    float mn = fminf(fminf(fminf(c4.x, c4.y), fminf(c4.z, c4.w)), fminf(fminf(r4.x, r4.y), fminf(r4.z, r4.w)));
    mx = warp_max(mx);
    mn = -warp_max(-mn);
    return mx / fmaxf(mn, vc.var_min);
  };

  // pass 0: row variances of the initial C = T (needed by I_best <- Imb(C), line 7); the row means mu_c are the
  // pivots of the later passes, and decide whether this tile needs them
  row_partials(std::false_type{}, 0.f);
  __syncthreads();
  bool off = false;
  if (tid < 128) {
    float s1 = 0.f, s2 = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) { s1 += sm.part[w][0][tid]; s2 += sm.part[w][1][tid]; }
    const float mean = s1 * inv_n;
    const float var = fmaxf(fmaf(-mean, mean, s2 * inv_n), 0.f);
    sm.mu[tid] = mean; sm.rvh[0][tid] = var; sm.Lrh[0][tid] = 0.f;
    off = mean * mean > 16.f * var;          // |mean| > 4 std: E[u^2] - E[u]^2 starts losing digits
  }
  const bool piv = __syncthreads_or(off);    // CTA-uniform
  if (piv) {   // redo pass 0 centred on mu (b = 1: exactly mean-free)
    row_partials(std::true_type{}, 1.f);
    __syncthreads();
    if (tid < 128) sm.rvh[0][tid] = row_variance_own();
    __syncthreads();
  }

  // The iterations, compiled twice: the plain form and the pivoted one (tiles with large channel offsets); a tile
  // runs one of them, so the plain form carries none of the pivot's code in its loop.
  auto varn_loop = [&](auto piv_tag) {
    constexpr bool PIV = decltype(piv_tag)::value;
    for (int k = 1; k <= vc.iters + 1; ++k) {
      const bool update = (k <= vc.iters);
      // ---- column half-step (lines 10-12): statistics of a_c T over channels ----
      {
        float v[16];
        {
          float2 s1[8], s2[8];
  #pragma unroll
          for (int i = 0; i < 8; ++i) { s1[i] = f2(0.f, 0.f); s2[i] = f2(0.f, 0.f); }
  #pragma unroll
          for (int i = 0; i < 8; ++i)
  #pragma unroll
            for (int kp = 0; kp < 4; ++kp) {
              float2 u = mul2(x[i][kp], a2[kp]);
              s1[i] = add2(s1[i], u);
              s2[i] = fma2(u, u, s2[i]);
            }
  #pragma unroll
          for (int i = 0; i < 8; ++i) { v[i] = s1[i].x + s1[i].y; v[8 + i] = s2[i].x + s2[i].y; }
        }
        float mine = xreduce16(v, li, OpAdd());
        float other = __shfl_xor_sync(0xffffffffu, mine, 8);
        const float s1t = (li & 8) ? other : mine, s2t = (li & 8) ? mine : other;
        const float mean = s1t * inv_n;
        const float var = fmaxf(fmaf(-mean, mean, s2t * inv_n), 0.f) * (b_own * b_own);
        if (li < 8) { sm.cvh[k - 1][tok_own] = var; sm.Lch[k - 1][tok_own] = Lc; }
        if (update) {
          const float vcl = fminf(fmaxf(var, vc.var_min), vc.var_max);
          Lc = fminf(fmaxf(fmaf(0.34657359027997264f, fast_log2(vcl), Lc), vc.log_lo), vc.log_hi);   // + 0.5 ln v
          b_own = fast_exp2(-1.4426950408889634f * Lc);                                               // e^-Lc
          if (li < 8) sm.b[tok_own] = b_own;
          __syncwarp();
          reload_b();
        }
      }
      // ---- row half-step (lines 13-15) --------------------------------------------
      // pivot scale bbar = mean_t b_t (tiles with large channel offsets only): in the first three iterations (b jumps
      // from 1 to 1 / S_c, then still moves by per cents) it is taken fresh, at the price of one more CTA barrier; later
      // it is the value warp 4 left during the previous iteration's row phase (one column update old: b then moves by
      // < 1e-3 per iteration)
      if (update) {
        if constexpr (PIV) {
          float bbar;
          if (k <= 3) {
            __syncthreads();
            const float4 b4 = reinterpret_cast<const float4*>(sm.b)[lane];
            bbar = warp_sum((b4.x + b4.y) + (b4.z + b4.w)) * inv_n;
          } else {
            bbar = sm.bbar;
          }
          row_partials(std::true_type{}, bbar);
        } else {
          row_partials(std::false_type{}, 0.f);
        }
      }
      __syncthreads();
      if (update) {
        if (PIV && warp == 4) {   // (idle in this phase) mean of the b the column half-step of this iteration left
          const float4 b4 = reinterpret_cast<const float4*>(sm.b)[lane];
          const float s = warp_sum((b4.x + b4.y) + (b4.z + b4.w)) * inv_n;
          if (lane == 0) sm.bbar = s;
        }
        if (tid < 128) {
          const float var = row_variance_own();
          const float vcl = fminf(fmaxf(var, vc.var_min), vc.var_max);
          const float Lr_new = fminf(fmaxf(fmaf(0.34657359027997264f, fast_log2(vcl), Lr), vc.log_lo), vc.log_hi);
          const float a_new = fast_exp2(-1.4426950408889634f * Lr_new);
          const float ratio = a_new * fast_exp2(1.4426950408889634f * Lr);   // a_new / a_old
          sm.rvh[k][tid] = var * ratio * ratio;  // row variance after rescaling the row
          sm.Lrh[k][tid] = Lr_new;
          sm.a[tid] = a_new;
          Lr = Lr_new; a_own = a_new;
        }
        __syncthreads();
        reload_a();
      }
    }
  };
  if (piv) varn_loop(std::true_type{}); else varn_loop(std::false_type{});

  // ---- best iterate (lines 7, 18): I_k = Imb(C_k), keep the last k with I_k <= min of the earlier ones
  __syncthreads();
  for (int k = warp; k <= vc.iters; k += 8) {
    const float imb = imbalance(k);
    if (lane == 0) {
      sm.imb[k] = imb;
      if (dbg.imb) dbg.imb[tile_idx * (KVARN_MAX_ITERS + 1) + k] = imb;
    }
  }
  __syncthreads();
  int k_best = 0;
  {
    float I_best = sm.imb[0];
    for (int k = 1; k <= vc.iters; ++k) {
      const float imb = sm.imb[k];
      if (imb <= I_best) { I_best = imb; k_best = k; }
    }
  }
  // ---- best scales (line 24): T_bal = T / S_c* / S_r* ----------------------------
  // aux_round = 1: the second scale (K: S_c per token, V: S_r per channel) balances the tile with its STORED value
  const bool rb = vc.aux_round != 0;
  if (li < 8) {
    const float L = sm.Lch[k_best][tok_own], S = expf(L);
    sm.Sc[tok_own] = S;
    sm.b[tok_own] = (rb && kind == KVARN_KIND_K) ? 1.f / e4m3_to_f32(f32_to_e4m3(S)) : expf(-L);
  }
  if (tid < 128) {
    const float L = sm.Lrh[k_best][tid], S = expf(L);
    sm.Sr[tid] = S;
    sm.a[tid] = (rb && kind == KVARN_KIND_V) ? 1.f / e4m3_to_f32(f32_to_e4m3(S)) : expf(-L);
  }
  __syncthreads();
  reload_a();
  reload_b();
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const float2 bb = f2(b[i], b[i]);
#pragma unroll
    for (int kp = 0; kp < 4; ++kp) x[i][kp] = mul2(mul2(x[i][kp], a2[kp]), bb);
  }

  // ---- Q3 + Q4: RTN group statistics, aux values ---------------------------------
  float inv_s[8], zz[8];  // of own channels (K) or own tokens (V)
  // group parameters from (mn, mx) and the absorbed Sinkhorn scale: pre-storage s1, the step the codes use
  // (1 / step in inv) and the zero-point the codes use (zc; zf = before FP16 rounding)
  auto group_params = [&](const float mn, const float mx, const float absorbed, float& s1, float& inv, float& zf, float& zc) {
    const float rng = mx - mn;
    const float s = (rng < 1e-12f) ? 1.f : rng / (float)LV;
    s1 = s * absorbed;
    if (rb) {
      const float s1q = e4m3_to_f32(f32_to_e4m3(s1));
      const float su = s1q > 0.f ? s1q / absorbed : s;
      zf = mn / su; zc = f16_bits_to_f32(f32_to_f16_bits(zf)); inv = 1.f / su;
    } else {
      zf = mn / s; zc = zf; inv = 1.f / s;
    }
  };
  // code = rint(x / step - z) by the magic-number add; with the stored parameters the value can leave [0, LV]
  const float2 magic = f2(RTN_MAGIC, RTN_MAGIC), nmagic = f2(-RTN_MAGIC, -RTN_MAGIC);
  auto rtn2 = [&](const float2 xv, const float2 is, const float2 nz) -> float2 {
    float2 q = add2(add2(fma2(xv, is, nz), magic), nmagic);
    if (rb) { q.x = fminf(fmaxf(q.x, 0.f), (float)LV); q.y = fminf(fmaxf(q.y, 0.f), (float)LV); }
    return q;
  };
  if (kind == KVARN_KIND_K) {
    // group = channel over the 128 tokens: min / max across warps through smem
    float mnv[8], mxv[8];
#pragma unroll
    for (int kp = 0; kp < 4; ++kp) {
      float mn0 = x[0][kp].x, mx0 = mn0, mn1 = x[0][kp].y, mx1 = mn1;
#pragma unroll
      for (int i = 1; i < 8; ++i) {
        mn0 = fminf(mn0, x[i][kp].x); mx0 = fmaxf(mx0, x[i][kp].x);
        mn1 = fminf(mn1, x[i][kp].y); mx1 = fmaxf(mx1, x[i][kp].y);
      }
      mnv[2 * kp] = mn0; mnv[2 * kp + 1] = mn1; mxv[2 * kp] = mx0; mxv[2 * kp + 1] = mx1;
    }
    float keep[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const float send = lj ? mnv[j] : mxv[j];
      const float got = __shfl_xor_sync(0xffffffffu, send, 16);
      keep[j] = lj ? fmaxf(mxv[j], got) : fminf(mnv[j], got);
    }
    float4* dst = reinterpret_cast<float4*>(&sm.part[warp][lj][c0]);
    dst[0] = make_float4(keep[0], keep[1], keep[2], keep[3]);
    dst[1] = make_float4(keep[4], keep[5], keep[6], keep[7]);
    __syncthreads();
    if (tid < 128) {
      float mn = sm.part[0][0][tid], mx = sm.part[0][1][tid];
#pragma unroll
      for (int w = 1; w < 8; ++w) { mn = fminf(mn, sm.part[w][0][tid]); mx = fmaxf(mx, sm.part[w][1][tid]); }
      float s1, inv, z, zc;
      group_params(mn, mx, sm.Sr[tid], s1, inv, z, zc);
      sm.inv_s[tid] = inv; sm.z[tid] = zc;
      const float s2 = sm.Sc[tid];  // K: s1 per channel, s2 per token
      const int kp = kaux_of_elem(BITS, tid);  // K records keep s1, z in B-operand builder order
      sm.rec[s1_off(BITS) + kp] = f32_to_e4m3(s1);
      sm.rec[s2_off(BITS) + slot_of_token(BITS, tid)] = f32_to_e4m3(s2);   // per-token arrays: MMA row-slot order
      reinterpret_cast<uint16_t*>(&sm.rec[z_off(BITS)])[kp] = f32_to_f16_bits(z);
      if (dbg.aux) {
        float* o = dbg.aux + tile_idx * 384;
        o[tid] = s1; o[128 + tid] = s2; o[256 + tid] = z;
      }
    }
    __syncthreads();
    const float4* pi = reinterpret_cast<const float4*>(&sm.inv_s[c0]);
    const float4* pz = reinterpret_cast<const float4*>(&sm.z[c0]);
    float4 i0 = pi[0], i1 = pi[1], z0 = pz[0], z1 = pz[1];
    inv_s[0] = i0.x; inv_s[1] = i0.y; inv_s[2] = i0.z; inv_s[3] = i0.w;
    inv_s[4] = i1.x; inv_s[5] = i1.y; inv_s[6] = i1.z; inv_s[7] = i1.w;
    zz[0] = z0.x; zz[1] = z0.y; zz[2] = z0.z; zz[3] = z0.w;
    zz[4] = z1.x; zz[5] = z1.y; zz[6] = z1.z; zz[7] = z1.w;
    // codes: row per token, channel c at bit BITS*(c%..) -- natural little-endian order.
    // code = rint(x / s - z) by the magic-number add (RNE, like rintf); x lies inside [mn, mx] of its
    // group, so x / s - z is within rounding error of [0, LV] and needs no clamp.  The 8 codes of a
    // thread are packed by exact float accumulation sum code_j 2^(BITS j) (< 2^16 per accumulator).
    float2 is2[4], nz2[4];
#pragma unroll
    for (int kp = 0; kp < 4; ++kp) { is2[kp] = f2(inv_s[2 * kp], inv_s[2 * kp + 1]); nz2[kp] = f2(-zz[2 * kp], -zz[2 * kp + 1]); }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int slot = slot_of_token(BITS, t0 + i);
      if (BITS == 2) {
        float2 acc = f2(0.f, 0.f);
#pragma unroll
        for (int kp = 0; kp < 4; ++kp) {
          const float2 q = rtn2(x[i][kp], is2[kp], nz2[kp]);
          acc = fma2(q, f2((float)(1 << (4 * kp)), (float)(4 << (4 * kp))), acc);
        }
        *reinterpret_cast<uint16_t*>(&sm.rec[code_off(2, slot, 2 * li)]) = (uint16_t)__float2uint_rn(acc.x + acc.y);
      } else {
        float2 lo = f2(0.f, 0.f), hi = f2(0.f, 0.f);
#pragma unroll
        for (int kp = 0; kp < 2; ++kp) {
          const float2 q0 = rtn2(x[i][kp], is2[kp], nz2[kp]);
          const float2 q1 = rtn2(x[i][kp + 2], is2[kp + 2], nz2[kp + 2]);
          const float2 wgt = f2((float)(1 << (8 * kp)), (float)(16 << (8 * kp)));
          lo = fma2(q0, wgt, lo);
          hi = fma2(q1, wgt, hi);
        }
        *reinterpret_cast<uint32_t*>(&sm.rec[code_off(4, slot, 4 * li)]) =
            __float2uint_rn(lo.x + lo.y) | (__float2uint_rn(hi.x + hi.y) << 16);
      }
    }
  } else {
    // group = token over the 128 channels: min / max inside the half-warp
    float v[16];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      float mn = fminf(x[i][0].x, x[i][0].y), mx = fmaxf(x[i][0].x, x[i][0].y);
#pragma unroll
      for (int kp = 1; kp < 4; ++kp) {
        mn = fminf(mn, fminf(x[i][kp].x, x[i][kp].y));
        mx = fmaxf(mx, fmaxf(x[i][kp].x, x[i][kp].y));
      }
      v[i] = mn; v[8 + i] = -mx;
    }
    float mine = xreduce16(v, li, OpMin());
    float other = __shfl_xor_sync(0xffffffffu, mine, 8);
    const float mn = (li & 8) ? other : mine, mx = -((li & 8) ? mine : other);
    float s1, inv, z, zc;
    group_params(mn, mx, sm.Sc[tok_own], s1, inv, z, zc);   // V: s1 per token
    if (li < 8) {
      sm.inv_s[tok_own] = inv; sm.z[tok_own] = zc;
      const int slot = slot_of_token(BITS, tok_own);
      sm.rec[s1_off(BITS) + slot] = f32_to_e4m3(s1);
      reinterpret_cast<uint16_t*>(&sm.rec[z_off(BITS)])[slot] = f32_to_f16_bits(z);
      if (dbg.aux) { float* o = dbg.aux + tile_idx * 384; o[tok_own] = s1; o[256 + tok_own] = z; }
    }
    if (tid < 128) {
      const float s2 = sm.Sr[tid];  // V: s2 per channel
      sm.rec[s2_off(BITS) + tid] = f32_to_e4m3(s2);
      if (dbg.aux) dbg.aux[tile_idx * 384 + 128 + tid] = s2;
    }
    __syncwarp();
    const float4* pi = reinterpret_cast<const float4*>(&sm.inv_s[t0]);
    const float4* pz = reinterpret_cast<const float4*>(&sm.z[t0]);
    float4 i0 = pi[0], i1 = pi[1], z0 = pz[0], z1 = pz[1];
    inv_s[0] = i0.x; inv_s[1] = i0.y; inv_s[2] = i0.z; inv_s[3] = i0.w;
    inv_s[4] = i1.x; inv_s[5] = i1.y; inv_s[6] = i1.z; inv_s[7] = i1.w;
    zz[0] = z0.x; zz[1] = z0.y; zz[2] = z0.z; zz[3] = z0.w;
    zz[4] = z1.x; zz[5] = z1.y; zz[6] = z1.z; zz[7] = z1.w;
    // codes: row per CHANNEL, token t at bit BITS*(t%..) of the row (rounding and packing as for K)
    float2 lo[4], hi[4];
#pragma unroll
    for (int kp = 0; kp < 4; ++kp) { lo[kp] = f2(0.f, 0.f); hi[kp] = f2(0.f, 0.f); }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const float2 is2 = f2(inv_s[i], inv_s[i]), nz2 = f2(-zz[i], -zz[i]);
      const float wv = BITS == 2 ? (float)(1 << (2 * i)) : (float)(1 << (4 * (i & 3)));
      const float2 wgt = f2(wv, wv);
#pragma unroll
      for (int kp = 0; kp < 4; ++kp) {
        const float2 q = rtn2(x[i][kp], is2, nz2);
        if (BITS == 2 || i < 4) lo[kp] = fma2(q, wgt, lo[kp]);
        else hi[kp] = fma2(q, wgt, hi[kp]);
      }
    }
#pragma unroll
    for (int kp = 0; kp < 4; ++kp) {
      if (BITS == 2) {
        *reinterpret_cast<uint16_t*>(&sm.rec[code_off(2, c0 + 2 * kp, 2 * (2 * warp + lj))]) = (uint16_t)__float2uint_rn(lo[kp].x);
        *reinterpret_cast<uint16_t*>(&sm.rec[code_off(2, c0 + 2 * kp + 1, 2 * (2 * warp + lj))]) = (uint16_t)__float2uint_rn(lo[kp].y);
      } else {
        *reinterpret_cast<uint32_t*>(&sm.rec[code_off(4, c0 + 2 * kp, 4 * (2 * warp + lj))]) =
            __float2uint_rn(lo[kp].x) | (__float2uint_rn(hi[kp].x) << 16);
        *reinterpret_cast<uint32_t*>(&sm.rec[code_off(4, c0 + 2 * kp + 1, 4 * (2 * warp + lj))]) =
            __float2uint_rn(lo[kp].y) | (__float2uint_rn(hi[kp].y) << 16);
      }
    }
  }
  if (dbg.k_best && tid == 0) dbg.k_best[tile_idx] = k_best;
  __syncthreads();

  // ---- Q5: write the record (coalesced 16-byte stores) ----------------------------
  {
    const uint4* src = reinterpret_cast<const uint4*>(sm.rec);
    uint4* dst = reinterpret_cast<uint4*>(rec_out);
    constexpr int NV = record_bytes(BITS) / 16;
    for (int i = tid; i < NV; i += 256) dst[i] = src[i];
  }
}

// Load rows t0..t0+7, channels c0..c0+7 of a tile into the register layout.
template <typename In>
__device__ __forceinline__ void load_row8(const In* __restrict__ row, float2 (&xr)[4]);

template <>
__device__ __forceinline__ void load_row8<__nv_bfloat16>(const __nv_bfloat16* __restrict__ row,
                                                         float2 (&xr)[4]) {
  const uint4 v = __ldg(reinterpret_cast<const uint4*>(row));
  const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int kp = 0; kp < 4; ++kp)
    xr[kp] = make_float2(__uint_as_float(w[kp] << 16), __uint_as_float(w[kp] & 0xffff0000u));
}
template <>
__device__ __forceinline__ void load_row8<float>(const float* __restrict__ row, float2 (&xr)[4]) {
  const float4 v0 = __ldg(reinterpret_cast<const float4*>(row));
  const float4 v1 = __ldg(reinterpret_cast<const float4*>(row) + 1);
  xr[0] = make_float2(v0.x, v0.y); xr[1] = make_float2(v0.z, v0.w);
  xr[2] = make_float2(v1.x, v1.y); xr[3] = make_float2(v1.z, v1.w);
}

}  // namespace kvarn

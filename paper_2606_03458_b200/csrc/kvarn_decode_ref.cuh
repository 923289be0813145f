// kvarn_decode_attention, CUDA-core version ("ref" path): split-K over chunks,
// every warp streams whole chunks with scalar FMAs.  It is the simple, easily
// audited implementation the tensor-core path is checked against on the GPU and
// the fallback for shapes that path does not cover.  SURVEY 8(a) rows D1-D7.
//
//   D1  q' = (q H / sqrt(128)) * sm_scale * log2(e)          (online Q transform)
//   D3  qt[h,c] = q'[h,c] s1[c];  beta[h] = sum_c qt[h,c] z[c]
//       logit[h,t] = s2[t] (sum_c qt[h,c] code[t,c] + beta[h])          (Eq. 1)
//   D4  online softmax in the log2 domain
//   D5  pt[h,t] = p[h,t] s1v[t];  a[h,c] = sum_t pt[h,t] codeV[t,c] + sum_t pt[h,t] zv[t]
//       acc_rot[h,c] += s2v[c] a[h,c]
//   D6  residual tokens: raw bf16 K/V in the un-rotated space
//   D7  merge splits (log-sum-exp), out = (acc_rot H / sqrt(128) + acc_res) / l
#pragma once

#include "kvarn_common.cuh"

namespace kvarn {

constexpr int WS_STRIDE = 260;  // floats per (b, hq, split): m, l, pad, pad, acc_rot[128], acc_res[128]

struct DecodeArgs {
  const uint8_t* k_records;
  const uint8_t* v_records;
  const void* k_resid;
  const void* v_resid;
  const int32_t* seq_lens;
  const void* q;
  void* out;
  float* ws;
  int B, Hkv, Hq, max_chunks, splits;
  float q_scale;  // sm_scale * log2(e)
  int rotate_k, rotate_v, out_dtype;
};

template <typename T> __device__ __forceinline__ float ld_in(const T* p);
template <> __device__ __forceinline__ float ld_in<float>(const float* p) { return *p; }
template <> __device__ __forceinline__ float ld_in<__nv_bfloat16>(const __nv_bfloat16* p) { return __bfloat162float(*p); }

template <int BITS, int GQ, typename InT>
__global__ void __launch_bounds__(128)
decode_partial_ref_kernel(const DecodeArgs A) {
  constexpr int LV = (1 << BITS) - 1;
  constexpr int RB = record_bytes(BITS);
  constexpr int ROWB = row_bytes(BITS);
  constexpr int WPR = ROWB / 4;          // 32-bit words per code row
  constexpr int CPW = 32 / BITS;         // codes per word
  const int bh = blockIdx.x, b = bh / A.Hkv, h = bh % A.Hkv;
  const int split = blockIdx.y;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  __shared__ __align__(16) float q_rot[GQ][128];
  __shared__ __align__(16) float q_raw[GQ][128];
  __shared__ __align__(16) float wbuf[4][GQ][128];   // per warp: qt, then pt
  __shared__ __align__(16) float macc[GQ][WS_STRIDE];

  // ---- D1: q prep ---------------------------------------------------------------
  for (int hh = warp; hh < GQ; hh += 4) {
    const InT* qp = reinterpret_cast<const InT*>(A.q) + ((size_t)b * A.Hq + h * GQ + hh) * D + 4 * lane;
    float v[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) { v[j] = ld_in<InT>(qp + j) * A.q_scale; q_raw[hh][4 * lane + j] = v[j]; }
    if (A.rotate_k) {
      fwht128_lane4(v, lane);
#pragma unroll
      for (int j = 0; j < 4; ++j) v[j] *= 0.08838834764831845f;
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) q_rot[hh][4 * lane + j] = v[j];
  }
  __syncthreads();

  const int len = A.seq_lens[b];
  int n_chunks = len >> 7;
  if (n_chunks > A.max_chunks) n_chunks = A.max_chunks;
  const int resid = len & 127;
  const int per = (n_chunks + A.splits - 1) / A.splits;
  const int c_begin = split * per, c_end = min(n_chunks, c_begin + per);

  float m[GQ], l[GQ], acc_rot[4][GQ], acc_res[4][GQ];
#pragma unroll
  for (int hh = 0; hh < GQ; ++hh) {
    m[hh] = -INFINITY; l[hh] = 0.f;
#pragma unroll
    for (int j = 0; j < 4; ++j) { acc_rot[j][hh] = 0.f; acc_res[j][hh] = 0.f; }
  }
  float(*wb)[128] = wbuf[warp];

  for (int ci = c_begin + warp; ci < c_end; ci += 4) {
    const uint8_t* kr = A.k_records + ((size_t)bh * A.max_chunks + ci) * RB;
    const uint8_t* vr = A.v_records + ((size_t)bh * A.max_chunks + ci) * RB;
    // ---- D3: fold K scales into q ------------------------------------------------
    float beta[GQ];
    {
      const uint32_t s1w = *reinterpret_cast<const uint32_t*>(kr + s1_off(BITS) + 4 * lane);
      const uint2 zw = *reinterpret_cast<const uint2*>(kr + z_off(BITS) + 8 * lane);
      float s1[4], z[4];
      float2 t0 = e4m3x2_to_f32x2((uint16_t)(s1w & 0xffff)), t1 = e4m3x2_to_f32x2((uint16_t)(s1w >> 16));
      s1[0] = t0.x; s1[1] = t0.y; s1[2] = t1.x; s1[3] = t1.y;
      z[0] = f16_bits_to_f32(zw.x & 0xffff); z[1] = f16_bits_to_f32(zw.x >> 16);
      z[2] = f16_bits_to_f32(zw.y & 0xffff); z[3] = f16_bits_to_f32(zw.y >> 16);
      __syncwarp();
#pragma unroll
      for (int hh = 0; hh < GQ; ++hh) {
        float bsum = 0.f;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const float qt = q_rot[hh][4 * lane + j] * s1[j];
          wb[hh][4 * lane + j] = qt;
          bsum = fmaf(qt, z[j], bsum);
        }
        beta[hh] = warp_sum(bsum);
      }
      __syncwarp();
    }
    // ---- logits of tokens lane + 32 jt ---------------------------------------------
    float logit[4][GQ];
#pragma unroll
    for (int jt = 0; jt < 4; ++jt) {
      const int t = lane + 32 * jt;
      const uint32_t* row = reinterpret_cast<const uint32_t*>(kr + (size_t)t * ROWB);
      float acc[GQ];
#pragma unroll
      for (int hh = 0; hh < GQ; ++hh) acc[hh] = 0.f;
#pragma unroll 2
      for (int wi = 0; wi < WPR; ++wi) {
        const uint32_t w = row[wi];
#pragma unroll
        for (int e = 0; e < CPW; e += 4) {
          float cv[4];
#pragma unroll
          for (int j = 0; j < 4; ++j) cv[j] = (float)((w >> (BITS * (e + j))) & LV);
          const int c = wi * CPW + e;
#pragma unroll
          for (int hh = 0; hh < GQ; ++hh) {
            const float4 qv = *reinterpret_cast<const float4*>(&wb[hh][c]);
            acc[hh] = fmaf(cv[0], qv.x, acc[hh]); acc[hh] = fmaf(cv[1], qv.y, acc[hh]);
            acc[hh] = fmaf(cv[2], qv.z, acc[hh]); acc[hh] = fmaf(cv[3], qv.w, acc[hh]);
          }
        }
      }
      const float s2 = e4m3_to_f32(kr[s2_off(BITS) + t]);
#pragma unroll
      for (int hh = 0; hh < GQ; ++hh) logit[jt][hh] = s2 * (acc[hh] + beta[hh]);
    }
    // ---- D4: online softmax; D5 prep: pt = p * s1v, zterm ---------------------------
    float corr[GQ], zterm[GQ];
    __syncwarp();
    {
      float s1v[4], zv[4];
#pragma unroll
      for (int jt = 0; jt < 4; ++jt) {
        const int t = lane + 32 * jt;
        s1v[jt] = e4m3_to_f32(vr[s1_off(BITS) + t]);
        zv[jt] = f16_bits_to_f32(reinterpret_cast<const uint16_t*>(vr + z_off(BITS))[t]);
      }
#pragma unroll
      for (int hh = 0; hh < GQ; ++hh) {
        float mx = fmaxf(fmaxf(logit[0][hh], logit[1][hh]), fmaxf(logit[2][hh], logit[3][hh]));
        mx = warp_max(mx);
        const float m_new = fmaxf(m[hh], mx);
        corr[hh] = (m[hh] == -INFINITY) ? 0.f : exp2f(m[hh] - m_new);
        float ps = 0.f, zs = 0.f;
#pragma unroll
        for (int jt = 0; jt < 4; ++jt) {
          const float p = exp2f(logit[jt][hh] - m_new);
          ps += p;
          const float pt = p * s1v[jt];
          wb[hh][lane + 32 * jt] = pt;
          zs = fmaf(pt, zv[jt], zs);
        }
        l[hh] = l[hh] * corr[hh] + warp_sum(ps);
        zterm[hh] = warp_sum(zs);
        m[hh] = m_new;
      }
    }
    __syncwarp();
    // ---- D5: values, channels lane + 32 jc ------------------------------------------
#pragma unroll
    for (int jc = 0; jc < 4; ++jc) {
      const int c = lane + 32 * jc;
      const uint32_t* row = reinterpret_cast<const uint32_t*>(vr + (size_t)c * ROWB);
      float acc[GQ];
#pragma unroll
      for (int hh = 0; hh < GQ; ++hh) acc[hh] = 0.f;
#pragma unroll 2
      for (int wi = 0; wi < WPR; ++wi) {
        const uint32_t w = row[wi];
#pragma unroll
        for (int e = 0; e < CPW; e += 4) {
          float cv[4];
#pragma unroll
          for (int j = 0; j < 4; ++j) cv[j] = (float)((w >> (BITS * (e + j))) & LV);
          const int t = wi * CPW + e;
#pragma unroll
          for (int hh = 0; hh < GQ; ++hh) {
            const float4 pv = *reinterpret_cast<const float4*>(&wb[hh][t]);
            acc[hh] = fmaf(cv[0], pv.x, acc[hh]); acc[hh] = fmaf(cv[1], pv.y, acc[hh]);
            acc[hh] = fmaf(cv[2], pv.z, acc[hh]); acc[hh] = fmaf(cv[3], pv.w, acc[hh]);
          }
        }
      }
      const float s2v = e4m3_to_f32(vr[s2_off(BITS) + c]);
#pragma unroll
      for (int hh = 0; hh < GQ; ++hh)
        acc_rot[jc][hh] = fmaf(acc_rot[jc][hh], corr[hh], s2v * (acc[hh] + zterm[hh]));
    }
    __syncwarp();
  }

  // ---- D6: residual window (raw tokens, un-rotated space), last split, warp 0 ----------
  if (split == A.splits - 1 && warp == 0 && resid > 0) {
    const InT* kres = reinterpret_cast<const InT*>(A.k_resid) + (size_t)bh * G * D;
    const InT* vres = reinterpret_cast<const InT*>(A.v_resid) + (size_t)bh * G * D;
    float logit[4][GQ];
#pragma unroll
    for (int jt = 0; jt < 4; ++jt) {
      const int t = lane + 32 * jt;
      float acc[GQ];
#pragma unroll
      for (int hh = 0; hh < GQ; ++hh) acc[hh] = 0.f;
      if (t < resid) {
        const InT* row = kres + (size_t)t * D;
        for (int c = 0; c < D; c += 4) {
          float kv[4];
#pragma unroll
          for (int j = 0; j < 4; ++j) kv[j] = ld_in<InT>(row + c + j);
#pragma unroll
          for (int hh = 0; hh < GQ; ++hh) {
            const float4 qv = *reinterpret_cast<const float4*>(&q_raw[hh][c]);
            acc[hh] = fmaf(kv[0], qv.x, acc[hh]); acc[hh] = fmaf(kv[1], qv.y, acc[hh]);
            acc[hh] = fmaf(kv[2], qv.z, acc[hh]); acc[hh] = fmaf(kv[3], qv.w, acc[hh]);
          }
        }
      }
#pragma unroll
      for (int hh = 0; hh < GQ; ++hh) logit[jt][hh] = (t < resid) ? acc[hh] : -INFINITY;
    }
    float corr[GQ];
    __syncwarp();
#pragma unroll
    for (int hh = 0; hh < GQ; ++hh) {
      float mx = fmaxf(fmaxf(logit[0][hh], logit[1][hh]), fmaxf(logit[2][hh], logit[3][hh]));
      mx = warp_max(mx);
      const float m_new = fmaxf(m[hh], mx);
      corr[hh] = (m[hh] == -INFINITY) ? 0.f : exp2f(m[hh] - m_new);
      float ps = 0.f;
#pragma unroll
      for (int jt = 0; jt < 4; ++jt) {
        const float p = exp2f(logit[jt][hh] - m_new);  // exp2(-inf) = 0 for masked tokens
        ps += p;
        wb[hh][lane + 32 * jt] = p;
      }
      l[hh] = l[hh] * corr[hh] + warp_sum(ps);
      m[hh] = m_new;
    }
    __syncwarp();
#pragma unroll
    for (int jc = 0; jc < 4; ++jc) {
      const int c = lane + 32 * jc;
      float acc[GQ];
#pragma unroll
      for (int hh = 0; hh < GQ; ++hh) acc[hh] = 0.f;
      for (int t = 0; t < resid; ++t) {
        const float vv = ld_in<InT>(vres + (size_t)t * D + c);
#pragma unroll
        for (int hh = 0; hh < GQ; ++hh) acc[hh] = fmaf(wb[hh][t], vv, acc[hh]);
      }
#pragma unroll
      for (int hh = 0; hh < GQ; ++hh) {
        acc_rot[jc][hh] *= corr[hh];
        acc_res[jc][hh] = acc[hh];
      }
    }
  }

  // ---- merge the four warps, write the split partial ---------------------------------
  for (int w = 0; w < 4; ++w) {
    __syncthreads();
    if (warp != w) continue;
#pragma unroll
    for (int hh = 0; hh < GQ; ++hh) {
      float* dst = macc[hh];
      if (w == 0) {
        if (lane == 0) { dst[0] = m[hh]; dst[1] = l[hh]; }
#pragma unroll
        for (int j = 0; j < 4; ++j) { dst[4 + lane + 32 * j] = acc_rot[j][hh]; dst[132 + lane + 32 * j] = acc_res[j][hh]; }
      } else {
        const float m_old = dst[0], l_old = dst[1];
        const float m_new = fmaxf(m_old, m[hh]);
        const float so = (m_old == -INFINITY) ? 0.f : exp2f(m_old - m_new);
        const float sn = (m[hh] == -INFINITY) ? 0.f : exp2f(m[hh] - m_new);
        __syncwarp();
        if (lane == 0) { dst[0] = m_new; dst[1] = l_old * so + l[hh] * sn; }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          dst[4 + lane + 32 * j] = dst[4 + lane + 32 * j] * so + acc_rot[j][hh] * sn;
          dst[132 + lane + 32 * j] = dst[132 + lane + 32 * j] * so + acc_res[j][hh] * sn;
        }
      }
    }
  }
  __syncthreads();
  for (int hh = 0; hh < GQ; ++hh) {
    float* o = A.ws + (((size_t)b * A.Hq + h * GQ + hh) * A.splits + split) * WS_STRIDE;
    for (int i = threadIdx.x; i < WS_STRIDE; i += 128) o[i] = macc[hh][i];
  }
}

// D7: merge split partials, inverse Hadamard, normalise.  One warp per (b, q head).
__global__ void __launch_bounds__(32) decode_merge_kernel(const DecodeArgs A) {
  const int bq = blockIdx.x, lane = threadIdx.x;
  const float* base = A.ws + (size_t)bq * A.splits * WS_STRIDE;
  float mstar = -INFINITY;
  for (int s = 0; s < A.splits; ++s) mstar = fmaxf(mstar, base[(size_t)s * WS_STRIDE]);
  float L = 0.f, rot[4] = {0.f, 0.f, 0.f, 0.f}, res[4] = {0.f, 0.f, 0.f, 0.f};
  for (int s = 0; s < A.splits; ++s) {
    const float* p = base + (size_t)s * WS_STRIDE;
    const float ms = p[0];
    const float w = (ms == -INFINITY) ? 0.f : exp2f(ms - mstar);
    L = fmaf(w, p[1], L);
    const float4 r4 = *reinterpret_cast<const float4*>(p + 4 + 4 * lane);
    const float4 s4 = *reinterpret_cast<const float4*>(p + 132 + 4 * lane);
    rot[0] = fmaf(w, r4.x, rot[0]); rot[1] = fmaf(w, r4.y, rot[1]);
    rot[2] = fmaf(w, r4.z, rot[2]); rot[3] = fmaf(w, r4.w, rot[3]);
    res[0] = fmaf(w, s4.x, res[0]); res[1] = fmaf(w, s4.y, res[1]);
    res[2] = fmaf(w, s4.z, res[2]); res[3] = fmaf(w, s4.w, res[3]);
  }
  if (A.rotate_v) {
    fwht128_lane4(rot, lane);
#pragma unroll
    for (int j = 0; j < 4; ++j) rot[j] *= 0.08838834764831845f;
  }
  const float inv = (L > 0.f) ? 1.f / L : 0.f;
  float o[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) o[j] = (rot[j] + res[j]) * inv;
  if (A.out_dtype == KVARN_F32) {
    *reinterpret_cast<float4*>(reinterpret_cast<float*>(A.out) + (size_t)bq * D + 4 * lane) =
        make_float4(o[0], o[1], o[2], o[3]);
  } else {
    __nv_bfloat162 v0 = __floats2bfloat162_rn(o[0], o[1]), v1 = __floats2bfloat162_rn(o[2], o[3]);
    uint2 u;
    u.x = *reinterpret_cast<uint32_t*>(&v0); u.y = *reinterpret_cast<uint32_t*>(&v1);
    *reinterpret_cast<uint2*>(reinterpret_cast<__nv_bfloat16*>(A.out) + (size_t)bq * D + 4 * lane) = u;
  }
}

}  // namespace kvarn

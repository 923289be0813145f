// kvarn_decode_attention for sm_100a: split-K over 128-token chunks, the two
// g x 128 x 128 contractions of every chunk on the 5th-gen tensor cores
// (tcgen05.mma kind::i8, accumulators in TMEM), records staged by TMA bulk copies.
// SURVEY 8(a) rows D1-D7; DESIGN.md "Decode kernel".
//
//   D1  q' = (q H / sqrt(128)) * sm_scale * log2(e)                    (online Q transform)
//   D2  record (codes + aux) -> shared memory ring, cp.async.bulk + mbarrier
//   D3  qt[h,c] = q'[h,c] s1[c];  beta[h] = sum_c qt[h,c] z[c]
//       logit[h,t] = s2[t] (sum_c qt[h,c] code[t,c] + beta[h])          (Eq. 1)
//   D4  online softmax in the log2 domain
//   D5  pt[h,t] = p[h,t] s1v[t];  a[h,c] = sum_t pt[h,t] (codeV[t,c] + zv[t]);  acc[h,c] += s2v[c] a[h,c]
//   D6  residual window: raw tokens in the un-rotated space
//   D7  split partials -> workspace; the last CTA of a (sequence, KV head) merges them
//       (log-sum-exp), applies the inverse Hadamard and normalises.
//
// How the contractions reach the tensor cores without a dequantised tile
// ---------------------------------------------------------------------
// A operand (M = 128 rows, K = 128, u8) lives in TMEM: thread r owns row r
// (K tile: token r, V tile: channel r), reads the row's packed codes from the
// staged record and expands them with ONE LOP3 per four codes:
//     column(NCLS*w + j) = W[w] & (MASK0 << BITS*j)
// i.e. the code stays where it is inside its byte and therefore carries the
// factor cls = 2^(BITS*j).  The B operand compensates: the fixed-point value
// of qt (or pt) at that K position is multiplied by CLSMAX / cls before it is
// split into radix-256 digits (s8 digits for qt, u8 digits for pt).  Each digit
// plane is one B row, so one MMA yields, per token, the exact int32 sums
//     D[t][i*GP + h] = sum_k A[t,k] * digit_i(X[h,k])
// and  sum_c Q[h,c] code[t,c] = (sum_i 256^i D[t][i*GP+h]) / CLSMAX  exactly.
// The only rounding is the fixed-point conversion of qt (22 bits + sign relative
// to max_c |qt[h,c]|) and pt (18 bits relative to max_t s1v[t]); beta and the
// zero-point term of V use the SAME fixed-point values, so no cancellation
// error appears between the code term and the zero-point term.
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
  int32_t* ticket;  // [B*Hkv], zero between calls (self-resetting)
  const void* q;
  void* out;
  float* ws;
  int B, Hkv, Hq, g, max_chunks, splits;
  float q_scale;  // sm_scale * log2(e)
  int rotate_k, rotate_v, out_dtype;
};

// ------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  const uint32_t a = smem_u32(bar);
  uint32_t done;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done) : "r"(a), "r"(parity) : "memory");
  } while (!done);
}
// TMA bulk copy global -> shared (1-D), completion on an mbarrier
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

template <int NCOLS>
__device__ __forceinline__ void tmem_alloc(uint32_t* slot) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slot)), "n"(NCOLS) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
template <int NCOLS>
__device__ __forceinline__ void tmem_dealloc(uint32_t base) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "n"(NCOLS) : "memory");
}
// 32 lanes x 32 columns: thread i of the warp writes r[0..31] to columns taddr.. of its lane
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,"
      "%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};"
      ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
        "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]),
        "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]),
        "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31])
      : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, int32_t (&d)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(d[0]), "=r"(d[1]), "=r"(d[2]), "=r"(d[3]), "=r"(d[4]), "=r"(d[5]), "=r"(d[6]), "=r"(d[7]),
        "=r"(d[8]), "=r"(d[9]), "=r"(d[10]), "=r"(d[11]), "=r"(d[12]), "=r"(d[13]), "=r"(d[14]), "=r"(d[15])
      : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// D[tmem] (+)= A[tmem, u8] * B[smem desc]; int32 accumulate
__device__ __forceinline__ void umma_i8_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::i8 [%0], [%1], %2, %3, p;\n\t}"
      ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// ------------------------------------------------------------------ operand geometry
// B operand in shared memory: MN-major ("transposed"), no swizzle.  Canonical
// layout ((16,m),(8,k)) : ((1,SBO),(16,LBO)) bytes: the 16 N values of one K
// position are 16 contiguous bytes, 8 consecutive K positions are 16 bytes apart
// (one 128-byte core matrix), groups of 8 K positions LBO = 128 bytes apart, and
// a second panel of 16 N values (GP = 8) SBO = 2048 bytes further.  So panel p of
// the operand is a dense [128 K positions][16 bytes] array, and the 16 bytes of
// a K position are (head-major) the radix-256 digits of 4 heads:
//     byte 4*(h & 3) + i of panel (h >> 2)  =  digit i of head h,
// i.e. a thread that holds the 32-bit fixed-point value X of (head h, K position
// k) stores X itself -- no byte transposes.  D column n = 4*h + i.
constexpr int B_LBO = 128;
constexpr int B_SBO = 2048;
constexpr int B_KSTEP = 32 * 16;   // bytes per MMA K step (32 K positions)
__host__ __device__ constexpr int b_bytes(int n_rows) { return (n_rows / 16) * B_SBO; }

__device__ __forceinline__ uint64_t b_desc(uint32_t saddr) {
  return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)(B_LBO >> 4) << 16) | ((uint64_t)(B_SBO >> 4) << 32) | (1ull << 46);
}
// idesc (kind::i8): D = s32, A = u8 (K-major, TMEM), B = s8 (b_signed) or u8, MN-major, M = 128
__host__ __device__ constexpr uint32_t idesc_i8(int n, int b_signed) {
  return (2u << 4) | (0u << 7) | ((uint32_t)b_signed << 10) | (1u << 16) | ((uint32_t)(n >> 3) << 17) | ((128u >> 4) << 24);
}

template <typename T> __device__ __forceinline__ float ld_in(const T* p);
template <> __device__ __forceinline__ float ld_in<float>(const float* p) { return *p; }
template <> __device__ __forceinline__ float ld_in<__nv_bfloat16>(const __nv_bfloat16* p) { return __bfloat162float(*p); }

// 8 consecutive input elements -> floats
__device__ __forceinline__ void ld_in8(const float* p, float (&v)[8]) {
  const float4 a = *reinterpret_cast<const float4*>(p), b = *reinterpret_cast<const float4*>(p + 4);
  v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
}
__device__ __forceinline__ void ld_in8(const __nv_bfloat16* p, float (&v)[8]) {
  const uint4 u = *reinterpret_cast<const uint4*>(p);
  const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) { v[2 * i] = __uint_as_float(w[i] << 16); v[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u); }
}

// Reduce NV values per lane over the 32 lanes of a warp with the exchange
// ("transpose") scheme: every step halves the number of live values until one is
// left, then plain butterflies.  Returns the reduced value of index
// red_index<NV>(lane) -- every index is held by 32/NV lanes.
template <int NV> __device__ __forceinline__ int red_index(int lane) {
  if (NV == 8) return ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);
  if (NV == 4) return ((lane >> 4) & 1) * 2 + ((lane >> 3) & 1);
  if (NV == 2) return (lane >> 4) & 1;
  return 0;
}
template <int LIVE, int M, int NV, class Op>
__device__ __forceinline__ void warp_reduce_step(float (&v)[NV], int lane, Op op) {
  if constexpr (LIVE > 1) {
    const bool up = lane & M;
#pragma unroll
    for (int j = 0; j < LIVE / 2; ++j) {
      const float send = up ? v[j] : v[j + LIVE / 2];
      const float keep = up ? v[j + LIVE / 2] : v[j];
      v[j] = op(keep, __shfl_xor_sync(0xffffffffu, send, M));
    }
    warp_reduce_step<LIVE / 2, M / 2>(v, lane, op);
  } else if constexpr (M > 0) {
    v[0] = op(v[0], __shfl_xor_sync(0xffffffffu, v[0], M));
    warp_reduce_step<1, M / 2>(v, lane, op);
  }
}
template <int NV, class Op>
__device__ __forceinline__ float warp_reduce_multi(float (&v)[NV], int lane, Op op) {
  warp_reduce_step<NV, 16>(v, lane, op);
  return v[0];
}
struct RAdd { __device__ __forceinline__ float operator()(float a, float b) const { return a + b; } };
struct RMax { __device__ __forceinline__ float operator()(float a, float b) const { return fmaxf(a, b); } };

constexpr float MAGIC_F = 12582912.0f;       // 1.5 * 2^23: (x + MAGIC) rounds x to an integer (RNE) for |x| <= 2^22
constexpr int MAGIC_I = 0x4B400000;
constexpr float Q_FIX = 4194300.0f;          // 2^22: fixed-point scale of qt relative to max_c |qt[h,c]|
constexpr float P_FIX = 4194304.0f;          // 2^22: fixed-point scale of pt = p s1v <= 1

template <int BITS, int GP>
struct DecSmem {
  static constexpr int RB = record_bytes(BITS);
  static constexpr int STAGES = BITS == 2 ? 3 : 2;
  static constexpr int NB = GP * 4;           // N of both MMAs: 4 radix-256 digits per head (D column 4 h + i)
  alignas(128) uint8_t rec[STAGES][2][RB];     // [stage][K | V] records
  alignas(128) uint8_t bq[b_bytes(NB)];
  alignas(128) uint8_t bp[b_bytes(NB)];
  alignas(16) float qrot[GP][128];             // q' (rotated, scaled); later: merged acc_rot for the inverse Hadamard
  alignas(16) float qraw[GP][128];             // q * q_scale (un-rotated, for the residual window); later p of the residual
  alignas(16) float hs[GP][2];                 // per head: {scale, beta} of the current chunk
  alignas(16) float wmax[4][GP];               // per-warp partial maxima
  alignas(16) float wz[4][GP];                 // per-warp partial zero-point sums / l sums
  alignas(8) uint64_t full[STAGES];
  alignas(8) uint64_t mma_bar[2];              // QK^T done, PV done
  uint32_t tmem_base;
  int last_flag;
};

// Expand the packed codes of row r of a staged record into A-operand columns.
template <int BITS>
__device__ __forceinline__ void unpack_row(const uint8_t* codes, int r, uint32_t (&a)[32]) {
  constexpr int NSEG = row_bytes(BITS) / 16;
  constexpr int NCLS = 8 / BITS;
  constexpr uint32_t MASK0 = BITS == 2 ? 0x03030303u : 0x0F0F0F0Fu;
#pragma unroll
  for (int s = 0; s < NSEG; ++s) {
    const uint4 w4 = *reinterpret_cast<const uint4*>(codes + s * 2048 + r * 16);
    const uint32_t w[4] = {w4.x, w4.y, w4.z, w4.w};
#pragma unroll
    for (int q = 0; q < 4; ++q)
#pragma unroll
      for (int j = 0; j < NCLS; ++j) a[NCLS * (4 * s + q) + j] = w[q] & (MASK0 << (BITS * j));
  }
}

template <int BITS, int GP, typename InT>
__global__ void __launch_bounds__(128, GP == 4 ? 6 : 4) decode_tc_kernel(const DecodeArgs A) {
  using SM = DecSmem<BITS, GP>;
  constexpr int RB = SM::RB, STAGES = SM::STAGES, NB = SM::NB;
  constexpr int NCLS = 8 / BITS;
  constexpr float CLS_INV = BITS == 2 ? (1.f / 64.f) : (1.f / 16.f);  // 1 / CLSMAX
  constexpr int HPW = GP / 4;                                          // heads per warp in the B_q builder
  // TMEM columns: A operand (K tile, then V tile of the same chunk), D (logits, then values)
  constexpr uint32_t TM_A = 0, TM_D = 32, TM_COLS = 64;

  extern __shared__ __align__(128) uint8_t smem_raw[];
  SM& sm = *reinterpret_cast<SM*>(smem_raw);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int bh = blockIdx.x, b = bh / A.Hkv, hkv = bh - b * A.Hkv;
  const int split = blockIdx.y;
  const int g = A.g;

  // ---- chunk range of this split ----------------------------------------------------
  const int len = A.seq_lens[b];
  int n_chunks = len >> 7;
  if (n_chunks > A.max_chunks) n_chunks = A.max_chunks;
  const int resid = len & 127;
  const int per = (n_chunks + A.splits - 1) / A.splits;
  const int c_begin = min(n_chunks, split * per), c_end = min(n_chunks, c_begin + per);
  const int n_my = c_end - c_begin;
  const bool do_resid = (split == A.splits - 1) && resid > 0;

  const uint8_t* krec = A.k_records + ((size_t)bh * A.max_chunks + c_begin) * RB;
  const uint8_t* vrec = A.v_records + ((size_t)bh * A.max_chunks + c_begin) * RB;

  // ---- setup: barriers, TMEM, first TMA loads, q ------------------------------------
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < STAGES; ++s) mbar_init(&sm.full[s], 1);
    mbar_init(&sm.mma_bar[0], 1);
    mbar_init(&sm.mma_bar[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
#pragma unroll
    for (int s = 0; s < STAGES; ++s)
      if (s < n_my) {
        mbar_expect_tx(&sm.full[s], 2 * RB);
        bulk_g2s(sm.rec[s][0], krec + (size_t)s * RB, RB, &sm.full[s]);
        bulk_g2s(sm.rec[s][1], vrec + (size_t)s * RB, RB, &sm.full[s]);
      }
  }
  if (warp == 1 && n_my > 0) tmem_alloc<TM_COLS>(&sm.tmem_base);

  // D1: q' = (q H / sqrt(128)) * q_scale; heads >= g are zero
  for (int hh = warp; hh < GP; hh += 4) {
    float v[4] = {0.f, 0.f, 0.f, 0.f};
    if (hh < g) {
      const InT* qp = reinterpret_cast<const InT*>(A.q) + ((size_t)b * A.Hq + hkv * g + hh) * D + 4 * lane;
#pragma unroll
      for (int j = 0; j < 4; ++j) v[j] = ld_in<InT>(qp + j) * A.q_scale;
    }
    *reinterpret_cast<float4*>(&sm.qraw[hh][4 * lane]) = make_float4(v[0], v[1], v[2], v[3]);
    if (A.rotate_k) {
      fwht128_lane4(v, lane);
#pragma unroll
      for (int j = 0; j < 4; ++j) v[j] *= 0.08838834764831845f;
    }
    *reinterpret_cast<float4*>(&sm.qrot[hh][4 * lane]) = make_float4(v[0], v[1], v[2], v[3]);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();

  // B_q builder role: warp -> heads warp (+4); lane owns K positions lane + 32 r, r = 0..3, which
  // all sit in byte (lane & 3) of an A column of class j = (lane >> 2) & (NCLS - 1):
  //   2-bit  channel = 32 r + 16 (lane >> 4) + 4 (lane & 3) + ((lane >> 2) & 3)
  //   4-bit  channel = 32 r +  8 (lane >> 3) + 2 (lane & 3) + ((lane >> 2) & 1)
  float qreg[HPW][4];
  {
    const int cbase = BITS == 2 ? 16 * (lane >> 4) + 4 * (lane & 3) + ((lane >> 2) & 3)
                                : 8 * (lane >> 3) + 2 * (lane & 3) + ((lane >> 2) & 1);
#pragma unroll
    for (int u = 0; u < HPW; ++u)
#pragma unroll
      for (int r = 0; r < 4; ++r) qreg[u][r] = sm.qrot[warp + 4 * u][cbase + 32 * r];
  }
  // fixed-point value -> digits: X = (bits(f) - MAGIC_I) << shift, balanced:  (X + 0x80808080) ^ 0x80808080
  const int shift_q = BITS * (NCLS - 1 - ((lane >> 2) & (NCLS - 1)));
  const uint32_t mul_q = 1u << shift_q;
  const uint32_t add_q = 0x80808080u - ((uint32_t)MAGIC_I << shift_q);
  // token role (softmax): K position of token tid in a V code row, and its class shift
  const int kpos_t = BITS == 2 ? ((tid & ~15) | ((tid & 3) << 2) | ((tid >> 2) & 3))
                               : ((tid & ~7) | ((tid & 1) << 2) | ((tid >> 1) & 3));
  const int shift_p = BITS * (NCLS - 1 - (tid & (NCLS - 1)));
  const uint32_t mul_p = 1u << shift_p;
  const uint32_t add_p = 0u - ((uint32_t)MAGIC_I << shift_p);

  float m_run[GP], l_part[GP], acc[GP];
#pragma unroll
  for (int h = 0; h < GP; ++h) { m_run[h] = -INFINITY; l_part[h] = 0.f; acc[h] = 0.f; }

  uint32_t tmem = 0, taddr_w = 0;
  if (n_my > 0) { tmem = sm.tmem_base; taddr_w = tmem + ((uint32_t)(warp * 32) << 16); }
  const uint32_t bq_addr = smem_u32(sm.bq), bp_addr = smem_u32(sm.bp);

  for (int it = 0; it < n_my; ++it) {
    const int st = it % STAGES;
    const uint32_t par = it & 1;
    const uint8_t* kr = sm.rec[st][0];
    const uint8_t* vr = sm.rec[st][1];
    mbar_wait(&sm.full[st], (it / STAGES) & 1);

    // ---- phase A: K codes -> TMEM, B_q (digits of the fixed-point qt), beta -----------
    {
      uint32_t a[32];
      unpack_row<BITS>(kr, tid, a);
      tmem_st32(taddr_w + TM_A, a);
    }
    {
      // aux of the K record in builder order: s1[4 lane + r], z[4 lane + r] <-> K position lane + 32 r
      const uint32_t s1w = *reinterpret_cast<const uint32_t*>(kr + s1_off(BITS) + 4 * lane);
      const uint2 zw = *reinterpret_cast<const uint2*>(kr + z_off(BITS) + 8 * lane);
      const float2 s01 = e4m3x2_to_f32x2((uint16_t)(s1w & 0xffff)), s23 = e4m3x2_to_f32x2((uint16_t)(s1w >> 16));
      const float s1[4] = {s01.x, s01.y, s23.x, s23.y};
      const float2 z01 = __half22float2(*reinterpret_cast<const __half2*>(&zw.x));
      const float2 z23 = __half22float2(*reinterpret_cast<const __half2*>(&zw.y));
      const float z[4] = {z01.x, z01.y, z23.x, z23.y};
      float qt[HPW][4], amax[HPW], bsum[HPW];
#pragma unroll
      for (int u = 0; u < HPW; ++u) {
#pragma unroll
        for (int r = 0; r < 4; ++r) qt[u][r] = qreg[u][r] * s1[r];
        amax[u] = fmaxf(fmaxf(fabsf(qt[u][0]), fabsf(qt[u][1])), fmaxf(fabsf(qt[u][2]), fabsf(qt[u][3])));
        // beta uses the unrounded qt: it differs from the 22-bit fixed-point value by < 2^-23 max|qt|
        bsum[u] = fmaf(qt[u][0], z[0], fmaf(qt[u][1], z[1], fmaf(qt[u][2], z[2], qt[u][3] * z[3])));
      }
#pragma unroll
      for (int u = 0; u < HPW; ++u)   // non-negative floats order like their bit patterns
        amax[u] = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(amax[u])));
#pragma unroll
      for (int m = 16; m > 0; m >>= 1)
#pragma unroll
        for (int u = 0; u < HPW; ++u) bsum[u] += __shfl_xor_sync(0xffffffffu, bsum[u], m);
#pragma unroll
      for (int u = 0; u < HPW; ++u) {
        const int h = warp + 4 * u;
        const float inv = amax[u] > 0.f ? Q_FIX * __fdividef(1.f, amax[u]) : 0.f;
        uint8_t* dst = sm.bq + (h >> 2) * B_SBO + lane * 16 + 4 * (h & 3);
#pragma unroll
        for (int r = 0; r < 4; ++r) {
          const float f = fmaf(qt[u][r], inv, MAGIC_F);            // integer Q in the low mantissa bits
          const uint32_t X = (__float_as_uint(f) * mul_q + add_q) ^ 0x80808080u;   // balanced s8 digits of Q << shift
          *reinterpret_cast<uint32_t*>(dst + r * 512) = X;
        }
        if (lane == 0) {
          const float sc = amax[u] * (1.f / Q_FIX);
          sm.hs[h][0] = sc * CLS_INV;   // logit = s2 * (acc * scale + beta)
          sm.hs[h][1] = bsum[u];
        }
      }
    }
    tmem_st_wait();
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();                                                   // barrier 1
    if (tid == 0) {
      tc_fence_after();
      const uint64_t bd = b_desc(bq_addr);
#pragma unroll
      for (int ks = 0; ks < 4; ++ks)
        umma_i8_ts(tmem + TM_D, tmem + TM_A + 8 * ks, bd + (uint64_t)((B_KSTEP * ks) >> 4), idesc_i8(NB, 1), ks > 0);
      umma_commit(&sm.mma_bar[0]);
    }

    // ---- phase B: per-token / per-channel aux of this chunk (overlaps the QK^T MMA) -------
    const float s2t = e4m3_to_f32(kr[s2_off(BITS) + tid]);
    const float s1v = fmaxf(e4m3_to_f32(vr[s1_off(BITS) + tid]), 9.094947e-13f);   // 2^-40: a zero scale stays harmless
    const float zv = f16_bits_to_f32(reinterpret_cast<const uint16_t*>(vr + z_off(BITS))[tid]);
    const float s2v = e4m3_to_f32(vr[s2_off(BITS) + tid]) * (1.f / P_FIX);   // channel role
    // pt = p s1v = exp2(logit + log2 s1v - m): the running maximum is taken over the shifted logits,
    // so pt <= 1 and its fixed-point scale is a constant
    const float lam = __log2f(s1v), inv_s1v = __fdividef(1.f, s1v);

    mbar_wait(&sm.mma_bar[0], par);
    tc_fence_after();
    {
      uint32_t a[32];                      // V codes -> the same TMEM columns (the QK^T MMA is done with them)
      unpack_row<BITS>(vr, tid, a);
      tmem_st32(taddr_w + TM_A, a);
    }
    // ---- D3/D4: logits of token tid, online softmax ---------------------------------------
    float logit[GP];
    {
      int32_t dlo[16], dhi[16];
      tmem_ld16(taddr_w + TM_D, dlo);
      if (NB == 32) tmem_ld16(taddr_w + TM_D + 16, dhi);
      tmem_ld_wait();
#pragma unroll
      for (int h = 0; h < GP; ++h) {
        const int32_t* d = h < 4 ? &dlo[4 * h] : &dhi[4 * (h & 3)];
        const int x01 = d[1] * 256 + d[0];
        const int x23 = d[3] * 256 + d[2];
        const float a = fmaf(__int2float_rn(x23), 65536.f, __int2float_rn(x01));
        const float2 sb = *reinterpret_cast<const float2*>(sm.hs[h]);
        logit[h] = fmaf(s2t, fmaf(a, sb.x, sb.y), lam);
      }
    }
    {
      float v[GP];
#pragma unroll
      for (int h = 0; h < GP; ++h) v[h] = logit[h];
      const float r = warp_reduce_multi<GP>(v, lane, RMax());
      if ((lane & (32 / GP - 1)) == 0) sm.wmax[warp][red_index<GP>(lane)] = r;
    }
    __syncthreads();                                                   // barrier 2
    float corr[GP], zpart[GP];
    uint32_t X[GP];
#pragma unroll
    for (int h = 0; h < GP; ++h) {
      const float mc = fmaxf(fmaxf(sm.wmax[0][h], sm.wmax[1][h]), fmaxf(sm.wmax[2][h], sm.wmax[3][h]));
      const float m_new = fmaxf(m_run[h], mc);
      corr[h] = exp2f(m_run[h] - m_new);
      m_run[h] = m_new;
      const float pt = exp2f(logit[h] - m_new);
      l_part[h] = fmaf(l_part[h], corr[h], pt * inv_s1v);
      // D5 prep: fixed-point pt; its radix-256 digits are the bytes of X
      const float f = fmaf(pt, P_FIX, MAGIC_F);
      zpart[h] = (f - MAGIC_F) * zv;
      X[h] = __float_as_uint(f) * mul_p + add_p;
    }
    *reinterpret_cast<uint4*>(sm.bp + kpos_t * 16) = make_uint4(X[0], X[1], X[2], X[3]);
    if (GP == 8) *reinterpret_cast<uint4*>(sm.bp + B_SBO + kpos_t * 16) = make_uint4(X[GP - 4], X[GP - 3], X[GP - 2], X[GP - 1]);
    {
      const float r = warp_reduce_multi<GP>(zpart, lane, RAdd());
      if ((lane & (32 / GP - 1)) == 0) sm.wz[warp][red_index<GP>(lane)] = r;
    }
    tmem_st_wait();
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();                                                   // barrier 3
    if (tid == 0) {
      tc_fence_after();
      const uint64_t bd = b_desc(bp_addr);
#pragma unroll
      for (int ks = 0; ks < 4; ++ks)
        umma_i8_ts(tmem + TM_D, tmem + TM_A + 8 * ks, bd + (uint64_t)((B_KSTEP * ks) >> 4), idesc_i8(NB, 0), ks > 0);
      umma_commit(&sm.mma_bar[1]);
      // the record slot is free (all aux values are in registers): prefetch chunk it + STAGES
      if (it + STAGES < n_my) {
        mbar_expect_tx(&sm.full[st], 2 * RB);
        bulk_g2s(sm.rec[st][0], krec + (size_t)(it + STAGES) * RB, RB, &sm.full[st]);
        bulk_g2s(sm.rec[st][1], vrec + (size_t)(it + STAGES) * RB, RB, &sm.full[st]);
      }
    }
    float zsum[GP];
#pragma unroll
    for (int h = 0; h < GP; ++h) zsum[h] = (sm.wz[0][h] + sm.wz[1][h]) + (sm.wz[2][h] + sm.wz[3][h]);

    // ---- D5: channel tid of the value contraction ---------------------------------------------
    mbar_wait(&sm.mma_bar[1], par);
    tc_fence_after();
    {
      int32_t dlo[16], dhi[16];
      tmem_ld16(taddr_w + TM_D, dlo);
      if (NB == 32) tmem_ld16(taddr_w + TM_D + 16, dhi);
      tmem_ld_wait();
#pragma unroll
      for (int h = 0; h < GP; ++h) {
        const int32_t* d = h < 4 ? &dlo[4 * h] : &dhi[4 * (h & 3)];
        const int x01 = d[1] * 256 + d[0];
        const int x23 = d[3] * 256 + d[2];
        const float a = fmaf(__int2float_rn(x23), 65536.f, __int2float_rn(x01));
        acc[h] = fmaf(acc[h], corr[h], s2v * fmaf(a, CLS_INV, zsum[h]));
      }
    }
    tc_fence_before();
  }

  // ---- D6: residual window (raw tokens, un-rotated space) -------------------------------------
  float acc_res[GP];
#pragma unroll
  for (int h = 0; h < GP; ++h) acc_res[h] = 0.f;
  if (do_resid) {
    const InT* kres = reinterpret_cast<const InT*>(A.k_resid) + (size_t)bh * G * D;
    const InT* vres = reinterpret_cast<const InT*>(A.v_resid) + (size_t)bh * G * D;
    float logit[GP];
#pragma unroll
    for (int h = 0; h < GP; ++h) logit[h] = 0.f;
    if (tid < resid) {
      const InT* row = kres + (size_t)tid * D;
      for (int c = 0; c < D; c += 8) {
        float kv[8];
        ld_in8(row + c, kv);
#pragma unroll
        for (int h = 0; h < GP; ++h) {
          const float4 q0 = *reinterpret_cast<const float4*>(&sm.qraw[h][c]);
          const float4 q1 = *reinterpret_cast<const float4*>(&sm.qraw[h][c + 4]);
          float s = logit[h];
          s = fmaf(kv[0], q0.x, s); s = fmaf(kv[1], q0.y, s); s = fmaf(kv[2], q0.z, s); s = fmaf(kv[3], q0.w, s);
          s = fmaf(kv[4], q1.x, s); s = fmaf(kv[5], q1.y, s); s = fmaf(kv[6], q1.z, s); s = fmaf(kv[7], q1.w, s);
          logit[h] = s;
        }
      }
    } else {
#pragma unroll
      for (int h = 0; h < GP; ++h) logit[h] = -INFINITY;
    }
    {
      float v[GP];
#pragma unroll
      for (int h = 0; h < GP; ++h) v[h] = logit[h];
      const float r = warp_reduce_multi<GP>(v, lane, RMax());
      if ((lane & (32 / GP - 1)) == 0) sm.wmax[warp][red_index<GP>(lane)] = r;
    }
    __syncthreads();   // also: every thread is done reading qraw as q
    float p[GP];
#pragma unroll
    for (int h = 0; h < GP; ++h) {
      const float mc = fmaxf(fmaxf(sm.wmax[0][h], sm.wmax[1][h]), fmaxf(sm.wmax[2][h], sm.wmax[3][h]));
      const float m_new = fmaxf(m_run[h], mc);
      const float corr = exp2f(m_run[h] - m_new);
      m_run[h] = m_new;
      p[h] = exp2f(logit[h] - m_new);        // exp2(-inf) = 0 for masked tokens
      l_part[h] = fmaf(l_part[h], corr, p[h]);
      acc[h] *= corr;
    }
    __syncthreads();
#pragma unroll
    for (int h = 0; h < GP; ++h) sm.qraw[h][tid] = p[h];
    __syncthreads();
    for (int t0 = 0; t0 < resid; t0 += 8) {
      float vv[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) vv[j] = (t0 + j < resid) ? ld_in<InT>(vres + (size_t)(t0 + j) * D + tid) : 0.f;
#pragma unroll
      for (int h = 0; h < GP; ++h) {
        const float4 p0 = *reinterpret_cast<const float4*>(&sm.qraw[h][t0]);
        const float4 p1 = *reinterpret_cast<const float4*>(&sm.qraw[h][t0 + 4]);
        float s = acc_res[h];
        s = fmaf(p0.x, vv[0], s); s = fmaf(p0.y, vv[1], s); s = fmaf(p0.z, vv[2], s); s = fmaf(p0.w, vv[3], s);
        s = fmaf(p1.x, vv[4], s); s = fmaf(p1.y, vv[5], s); s = fmaf(p1.z, vv[6], s); s = fmaf(p1.w, vv[7], s);
        acc_res[h] = s;
      }
    }
  }

  // ---- l: reduce the per-thread partial sums ----------------------------------------------------
  __syncthreads();
  {
    float v[GP];
#pragma unroll
    for (int h = 0; h < GP; ++h) v[h] = l_part[h];
    const float r = warp_reduce_multi<GP>(v, lane, RAdd());
    if ((lane & (32 / GP - 1)) == 0) sm.wz[warp][red_index<GP>(lane)] = r;
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1 && n_my > 0) { tc_fence_after(); tmem_dealloc<64>(tmem); }
  float l_tot[GP];
#pragma unroll
  for (int h = 0; h < GP; ++h) l_tot[h] = (sm.wz[0][h] + sm.wz[1][h]) + (sm.wz[2][h] + sm.wz[3][h]);

  // ---- D7: partials -> workspace; last CTA of this (sequence, KV head) merges -------------------
  float* merged_rot = &sm.qrot[0][0];   // [GP][128]
  float Ltot[GP];
#pragma unroll
  for (int h = 0; h < GP; ++h) Ltot[h] = 0.f;
  if (A.splits > 1) {
#pragma unroll
    for (int h = 0; h < GP; ++h) {
      if (h < g) {
        float* o = A.ws + (((size_t)b * A.Hq + hkv * g + h) * A.splits + split) * WS_STRIDE;
        if (tid == 0) { o[0] = m_run[h]; o[1] = l_tot[h]; }
        o[4 + tid] = acc[h];
        o[132 + tid] = acc_res[h];
      }
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) {
      const int old = atomicAdd(&A.ticket[bh], 1);
      const int last = (old == A.splits - 1);
      if (last) A.ticket[bh] = 0;
      sm.last_flag = last;
    }
    __syncthreads();
    if (!sm.last_flag) return;
    __threadfence();
    // weights of the splits: warp w handles heads w, w+4; lane s handles splits s, s+32
    float* wsp = reinterpret_cast<float*>(sm.bq);   // [GP][64] split weights (B_q is dead by now)
    for (int h = warp; h < g; h += 4) {
      const float* base = A.ws + ((size_t)b * A.Hq + hkv * g + h) * A.splits * WS_STRIDE;
      const float m0 = lane < A.splits ? __ldcg(base + (size_t)lane * WS_STRIDE) : -INFINITY;
      const float m1 = lane + 32 < A.splits ? __ldcg(base + (size_t)(lane + 32) * WS_STRIDE) : -INFINITY;
      const float l0 = lane < A.splits ? __ldcg(base + (size_t)lane * WS_STRIDE + 1) : 0.f;
      const float l1 = lane + 32 < A.splits ? __ldcg(base + (size_t)(lane + 32) * WS_STRIDE + 1) : 0.f;
      const float mstar = warp_max(fmaxf(m0, m1));
      const float w0 = (m0 == -INFINITY) ? 0.f : exp2f(m0 - mstar);
      const float w1 = (m1 == -INFINITY) ? 0.f : exp2f(m1 - mstar);
      wsp[h * 64 + lane] = w0;
      wsp[h * 64 + lane + 32] = w1;
      const float L = warp_sum(fmaf(w0, l0, w1 * l1));
      if (lane == 0) sm.hs[h][1] = L;
    }
    __syncthreads();
#pragma unroll
    for (int h = 0; h < GP; ++h) {
      if (h < g) {
        const float* base = A.ws + ((size_t)b * A.Hq + hkv * g + h) * A.splits * WS_STRIDE + 4 + tid;
        float rot = 0.f, res = 0.f;
        int s = 0;
        for (; s + 4 <= A.splits; s += 4) {
          float r[4], e[4];
#pragma unroll
          for (int j = 0; j < 4; ++j) { r[j] = __ldcg(base + (size_t)(s + j) * WS_STRIDE); e[j] = __ldcg(base + (size_t)(s + j) * WS_STRIDE + 128); }
#pragma unroll
          for (int j = 0; j < 4; ++j) { const float w = wsp[h * 64 + s + j]; rot = fmaf(w, r[j], rot); res = fmaf(w, e[j], res); }
        }
        for (; s < A.splits; ++s) {
          const float w = wsp[h * 64 + s];
          rot = fmaf(w, __ldcg(base + (size_t)s * WS_STRIDE), rot);
          res = fmaf(w, __ldcg(base + (size_t)s * WS_STRIDE + 128), res);
        }
        Ltot[h] = sm.hs[h][1]; acc[h] = rot; acc_res[h] = res;
      }
    }
  } else {
#pragma unroll
    for (int h = 0; h < GP; ++h) Ltot[h] = l_tot[h];
  }
  __syncthreads();
#pragma unroll
  for (int h = 0; h < GP; ++h) {
    merged_rot[h * 128 + tid] = acc[h];
    sm.qraw[h][tid] = (Ltot[h] > 0.f) ? acc_res[h] : 0.f;
    if (tid == 0) sm.hs[h][0] = (Ltot[h] > 0.f) ? 1.f / Ltot[h] : 0.f;
  }
  __syncthreads();
  for (int hh = warp; hh < g; hh += 4) {
    float4 r4 = *reinterpret_cast<const float4*>(&merged_rot[hh * 128 + 4 * lane]);
    float v[4] = {r4.x, r4.y, r4.z, r4.w};
    if (A.rotate_v) {
      fwht128_lane4(v, lane);
#pragma unroll
      for (int j = 0; j < 4; ++j) v[j] *= 0.08838834764831845f;
    }
    const float4 s4 = *reinterpret_cast<const float4*>(&sm.qraw[hh][4 * lane]);
    const float inv = sm.hs[hh][0];
    const float o0 = (v[0] + s4.x) * inv, o1 = (v[1] + s4.y) * inv, o2 = (v[2] + s4.z) * inv, o3 = (v[3] + s4.w) * inv;
    const size_t off = ((size_t)b * A.Hq + hkv * g + hh) * D + 4 * lane;
    if (A.out_dtype == KVARN_F32) {
      *reinterpret_cast<float4*>(reinterpret_cast<float*>(A.out) + off) = make_float4(o0, o1, o2, o3);
    } else {
      __nv_bfloat162 v0 = __floats2bfloat162_rn(o0, o1), v1 = __floats2bfloat162_rn(o2, o3);
      uint2 u;
      u.x = *reinterpret_cast<uint32_t*>(&v0); u.y = *reinterpret_cast<uint32_t*>(&v1);
      *reinterpret_cast<uint2*>(reinterpret_cast<__nv_bfloat16*>(A.out) + off) = u;
    }
  }
}

}  // namespace kvarn

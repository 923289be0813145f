// Dense multi-token read path on the 5th-generation tensor cores (tcgen05 + TMEM): a block of query rows against the
// packed chunks of the cache (Fig. 4 pseudo-decode).  Used by kvarn_block_attention_dense
// for blocks with many (query token, head) rows per KV head; the raw windows (sink, residual, the block's own causal
// tokens) are left to decode_kernel_w (skip_chunks = 1, partial = 1) and everything is merged by merge_partials_kernel.
//
// One CTA = one (sequence, KV head), one tile of 128 query rows r = (token i, head h), one range of chunks; 9 warps in
// three roles that meet only through mbarriers: warps 4-7 expand the records (producers), one thread of warp 8 issues
// the MMAs, warps 0-3 own the softmax (thread = query row = TMEM lane).  While the softmax warps work on chunk i the
// producers already expand V of chunk i and K of chunk i + 1 and the tensor core runs QK^T of chunk i + 1.  Per chunk:
//   K record --TMA--> shared memory --128 threads--> Kt = code x s1[c] as fp16 (EXACT: a 2-/4-bit code times an E4M3
//     scale has <= 8 significant bits), K-major UMMA tile [token][channel], + two rows hi / lo of (s1 z)[c] for beta
//   S[r][t] = sum_c (q'_hi + q'_lo)[r][c] Kt[t][c]          tcgen05.mma kind::f16, M = 128, N = 144, K = 128, twice (hi, lo)
//   logit = s2[t] (S + beta_r) + log2 s1v[t];  online softmax per ROW inside one thread (TMEM lane = row)
//   Pt = p~ as fp16 (+ hi / lo of the zero-point sum as two extra K columns)
//   V record --> Vt = codeV x s2v[c] as fp16 (exact), [channel][token] (+ s2v[c] in the two extra K columns)
//   O[r][c] += sum_t Pt[r][t] Vt[c][t]                      tcgen05.mma, M = 128, N = 128, K = 144, accumulator in TMEM
// The accumulator is rescaled in TMEM (tcgen05.ld / st) only when a row's maximum rises.  Finally O is un-rotated
// (inverse Hadamard) and written as the partial {m, l, o[128]} of its rows.
//
// Precision: q' enters as two fp16 terms (22 bits), codes x scales exactly, beta through the same MMA; p~ is fp16
// relative to 2^-8 of the row's running maximum (so probabilities down to 2^-32 of it survive) and l is accumulated
// from the SAME rounded values; fp32 accumulation in TMEM.
#pragma once

#include "kvarn_decode.cuh"

namespace kvarn {

struct DenseArgs {
  const uint8_t* k_records;
  const uint8_t* v_records;
  const int32_t* seq_lens;
  const void* q;        // [B][n_q][Hq][128]
  float* parts;         // [splits][B * n_q * Hq][PART_STRIDE]
  int B, Hkv, Hq, g, max_chunks, n_sink, n_q, splits, n_tiles;
  float q_scale;
  int rotate_k, rotate_v;
};

constexpr int DN_KT = 128;                 // K extent of the QK^T tiles (channels)
constexpr int DN_KP = 144;                 // K extent of the PV tiles (128 tokens + 16: zero-point columns)
constexpr int DN_NS = 144;                 // N of the QK^T MMA (128 tokens + 16: beta rows)
constexpr int DN_KPH = 80;                 // K extent of one token half of p~ (64 tokens + 16: zero-point columns)

// byte offset of element (row r, column k) of a K-major, un-swizzled fp16 UMMA tile with KT columns:
// core matrices of 8 rows x 16 bytes, 128 B apart along K (LBO), (KT / 8) * 128 B apart along M / N (SBO)
__host__ __device__ constexpr int kmaj_off(int r, int k, int KT) {
  return (r >> 3) * ((KT >> 3) * 128) + (k >> 3) * 128 + (r & 7) * 16 + (k & 7) * 2;
}
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16) |
         ((uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32) | ((uint64_t)1 << 46);   // version 1, no swizzle
}
// kind::f16 instruction descriptor: D fp32, A / B fp16, both K-major, N >> 3 at bit 17, M >> 4 at bit 24
__host__ __device__ constexpr uint32_t umma_idesc_f16(int M, int N) {
  return (1u << 4) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void umma_f16(uint32_t d_tmem, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
               ::"r"(d_tmem), "l"(da), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                 "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]) : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&v)[16]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
               ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
                 "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// K position of element e (a channel of a K row / a token of a V row) inside the dense tiles: the fp16 expansion
// takes codes j and j + CPW / 2 of a packed word in one half2, so these two become neighbours along K.
template <int BITS> __host__ __device__ constexpr int dense_kpos(int e) {
  constexpr int CPW = 32 / BITS;
  return (e / CPW) * CPW + 2 * (e % (CPW / 2)) + ((e % CPW) / (CPW / 2));
}
template <int BITS> __host__ __device__ constexpr int dense_elem_of_kpos(int kp) {
  constexpr int CPW = 32 / BITS;
  return (kp / CPW) * CPW + ((kp % CPW) >> 1) + (kp & 1) * (CPW / 2);
}

template <int BITS>
struct DenseSmem {
  static constexpr int RB = record_bytes(BITS);
  alignas(1024) uint8_t qhi[128 * DN_KT * 2];      // q' (rotated, scaled), first fp16 term; later: staging of O (with qlo)
  alignas(1024) uint8_t qlo[128 * DN_KT * 2];      // second fp16 term
  alignas(1024) uint8_t kt[DN_NS * DN_KT * 2];     // rows 0..127: token rho(t); 128, 129: hi / lo of s1 z; 130..143: zero
  alignas(1024) uint8_t vt[128 * DN_KP * 2];       // rows: channels; columns 0..127 tokens (rho order), 128, 129: s2v, rest zero
  alignas(1024) uint8_t pt[2][128 * DN_KPH * 2];   // [token half] rows: query rows; columns 0..63 p~, 64, 65: hi / lo of zsum
  alignas(128) uint8_t rec_k[2][RB];               // [chunk parity]
  alignas(128) uint8_t rec_v[2][RB];
  alignas(16) __half2 s1h[64];                     // s1 of the K record as fp16 pairs in K-position order
  alignas(16) float2 aux_a[2][128];                // [chunk parity] per token (rho order): {s2, log2 s1v}
  alignas(16) float2 aux_b[2][128];                //                                       {1 / s1v, zv}
  alignas(16) float2 ml[128];                      // epilogue: {m, l} of the rows
  alignas(8) uint64_t full_k[2], full_v[2];        // TMA arrival [chunk parity]
  alignas(8) uint64_t bar_s, bar_o[2];             // MMA completion (tcgen05.commit): S ready, O of a token half accumulated
  alignas(8) uint64_t kt_full, vt_full;            // producers -> issuer (and softmax warps: aux) (256 arrivals each)
  alignas(8) uint64_t s_free, p_full[2];           // softmax warps -> issuer (256 / 128 arrivals)
  uint32_t tmem_base;
};

// the packed words of half `half` (K positions 64 half .. 64 half + 63) of the code row in slot `slot`
template <int BITS>
__device__ __forceinline__ void load_row_half(const uint8_t* codes, int slot, int half, uint32_t (&W)[2 * BITS]) {
  const int w = slot >> 5, mt = (slot >> 4) & 1, rho = (slot >> 3) & 1, g = slot & 7;
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    if constexpr (BITS == 2) {
      W[t] = *reinterpret_cast<const uint32_t*>(codes + w * 1024 + mt * 512 + (4 * g + t) * 16 + rho * 8 + 4 * half);
    } else {
      const uint2 v = *reinterpret_cast<const uint2*>(codes + w * 2048 + mt * 1024 + rho * 512 + (4 * g + t) * 16 + 8 * half);
      W[t] = v.x; W[4 + t] = v.y;
    }
  }
}

// Half a code row (64 codes) -> 64 fp16 values code * scale in K-position order, written as 8 units of 16 bytes of
// row `row` of a K-major tile with KT columns.  scale_tab: half2 per K-position pair (64 entries), or null: `sc` for all.
template <int BITS, bool TAB>
__device__ __forceinline__ void dequant_half(const uint32_t (&W)[2 * BITS], const __half2* scale_tab, __half2 sc,
                                             uint8_t* tile, int row, int KT, int half) {
  constexpr int CPW = 32 / BITS, PPW = CPW / 2;                 // codes, pairs per word
  constexpr uint32_t MASK = BITS == 2 ? 0x00030003u : 0x000F000Fu;
  const __half2 k1024 = __floats2half2_rn(1024.f, 1024.f);
  uint8_t* base = tile + (row >> 3) * ((KT >> 3) * 128) + (row & 7) * 16 + half * 1024;
  if (TAB) scale_tab += 32 * half;
#pragma unroll
  for (int u = 0; u < 8; ++u) {                                  // unit u: K positions 64 half + 8u .. + 7 = 4 pairs
    uint32_t o[4];
#pragma unroll
    for (int pp = 0; pp < 4; ++pp) {
      const int pair = 4 * u + pp;                               // pair index inside the half
      const int wi = pair / PPW, j = pair % PPW;
      uint32_t h = ((W[wi] >> (BITS * j)) & MASK) | 0x64006400u; // fp16 1024 + code, twice
      __half2 x = __hsub2(*reinterpret_cast<__half2*>(&h), k1024);
      x = __hmul2(x, TAB ? scale_tab[pair] : sc);
      o[pp] = *reinterpret_cast<uint32_t*>(&x);
    }
    *reinterpret_cast<uint4*>(base + u * 128) = make_uint4(o[0], o[1], o[2], o[3]);
  }
}

__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void producer_sync() { asm volatile("bar.sync 1, 256;" ::: "memory"); }
__device__ __forceinline__ void tmem_ld2(uint32_t taddr, uint32_t& a, uint32_t& b) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0,%1}, [%2];" : "=r"(a), "=r"(b) : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}



constexpr int DENSE_THREADS = 544;          // warps 0-7 softmax, 8-15 producers, 16 MMA issuer
constexpr int DENSE_SETS = 2;               // partial sets per CTA: one per token half (independent online softmax streams)

template <int BITS, typename InT>
__global__ void __launch_bounds__(DENSE_THREADS, 1) block_dense_kernel(const DenseArgs A) {
  using SM = DenseSmem<BITS>;
  constexpr int RB = SM::RB;
  constexpr uint32_t TMEM_COLS = 512;           // S: columns [0, 144), O of token half h: columns [256 + 128 h, 384 + 128 h)
  constexpr uint32_t O_COL = 256;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  SM& sm = *reinterpret_cast<SM*>(smem_raw);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = A.g;
  const int unit = blockIdx.x / A.n_tiles, rt = blockIdx.x - unit * A.n_tiles;     // (b, kv head), row tile
  const int b = unit / A.Hkv, hkv = unit - b * A.Hkv, split = blockIdx.y;
  const int len = A.seq_lens[b];
  const int body = len - min(len, A.n_sink);
  const int n_chunks = min(body >> 7, A.max_chunks);
  const int per = (n_chunks + A.splits - 1) / A.splits;
  const int c_begin = min(split * per, n_chunks), c_end = min(c_begin + per, n_chunks);
  const int n_my = c_end - c_begin;
  const int n_rows = A.n_q * g;                                                     // query rows of this (b, kv head)
  const uint8_t* krec = A.k_records + ((size_t)unit * A.max_chunks + c_begin) * RB;
  const uint8_t* vrec = A.v_records + ((size_t)unit * A.max_chunks + c_begin) * RB;

  // ---- setup: barriers, TMEM, first records, q ------------------------------------------------------------------
  if (tid == 256) {
    for (int s = 0; s < 2; ++s) { mbar_init(&sm.full_k[s], 1); mbar_init(&sm.full_v[s], 1); mbar_init(&sm.bar_o[s], 1); mbar_init(&sm.p_full[s], 128); }
    mbar_init(&sm.bar_s, 1);
    mbar_init(&sm.kt_full, 256); mbar_init(&sm.vt_full, 256); mbar_init(&sm.s_free, 256);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    for (int c = 0; c < 2 && c < n_my; ++c) {
      mbar_expect_tx(&sm.full_k[c], RB); bulk_g2s(sm.rec_k[c], krec + (size_t)c * RB, RB, &sm.full_k[c]);
      mbar_expect_tx(&sm.full_v[c], RB); bulk_g2s(sm.rec_v[c], vrec + (size_t)c * RB, RB, &sm.full_v[c]);
    }
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&sm.tmem_base)), "n"(TMEM_COLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  // zero the tiles once: rows / columns that are never rewritten (padding of N = 144 and of the K extents) stay zero
  for (int i = tid; i < (int)(sizeof(sm.kt) / 16); i += DENSE_THREADS) reinterpret_cast<uint4*>(sm.kt)[i] = make_uint4(0, 0, 0, 0);
  for (int i = tid; i < (int)(sizeof(sm.vt) / 16); i += DENSE_THREADS) reinterpret_cast<uint4*>(sm.vt)[i] = make_uint4(0, 0, 0, 0);
  for (int i = tid; i < (int)(sizeof(sm.pt) / 16); i += DENSE_THREADS) reinterpret_cast<uint4*>(sm.pt)[i] = make_uint4(0, 0, 0, 0);
  // q' = (q H / sqrt(128)) q_scale as two fp16 terms, columns in K-position order
  for (int r = warp; r < 128; r += DENSE_THREADS / 32) {
    const int R = rt * 128 + r;
    float v[4] = {0.f, 0.f, 0.f, 0.f};
    if (R < n_rows) {
      const int i = R / g, h = R - i * g;
      const size_t row = ((size_t)b * A.n_q + i) * A.Hq + hkv * g + h;
      const InT* qp = reinterpret_cast<const InT*>(A.q) + row * D + 4 * lane;
#pragma unroll
      for (int j = 0; j < 4; ++j) v[j] = ld_in<InT>(qp + j) * A.q_scale;
    }
    if (A.rotate_k) {
      fwht128_lane4(v, lane);
#pragma unroll
      for (int j = 0; j < 4; ++j) v[j] *= 0.08838834764831845f;
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int kp = dense_kpos<BITS>(4 * lane + j);
      const __half hi = __float2half_rn(v[j]);
      const __half lo = __float2half_rn(v[j] - __half2float(hi));
      *reinterpret_cast<__half*>(sm.qhi + kmaj_off(r, kp, DN_KT)) = hi;
      *reinterpret_cast<__half*>(sm.qlo + kmaj_off(r, kp, DN_KT)) = lo;
    }
  }
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = sm.tmem_base;
  constexpr uint32_t IDESC_S = umma_idesc_f16(128, DN_NS), IDESC_O = umma_idesc_f16(128, 128);
  constexpr uint32_t SBO_T = (DN_KT / 8) * 128, SBO_P = (DN_KP / 8) * 128, SBO_PH = (DN_KPH / 8) * 128;
  constexpr float P_OFF = 8.f;                  // p~ = 2^(logit - max + 8): probabilities down to 2^-32 of the maximum survive fp16
  float m_ref = -INFINITY, l_run = 0.f;         // softmax warps: reference exponent of the (row, token half), running l

  // Barrier phases: phase i of kt_full / vt_full / s_free / p_full / bar_s / bar_o belongs to chunk i (parity i & 1).  No
  // barrier completes phase i + 1 before every waiter of phase i has looked (a parity wait cannot tell i from i + 2):
  // the waits marked (*) below are there for that reason alone.
  if (warp >= 8 && warp < 16) {
    // =============================== producers: thread = (token | channel row, half of its codes) ====================
    const int pt = tid - 256, row = pt & 127, half = pt >> 7;
    const int rho_t = dense_kpos<BITS>(row), slot_t = slot_of_token(BITS, row);
    // chunk c: per-channel and per-token aux, then Kt; afterwards the K record of chunk c + 2 is requested
    auto expand_k = [&](int c) {
      const int st = c & 1;
      const uint32_t par_rec = (c >> 1) & 1;
      mbar_wait(&sm.full_k[st], par_rec);
      mbar_wait(&sm.full_v[st], par_rec);
      const uint8_t* kr = sm.rec_k[st];
      const uint8_t* vr = sm.rec_v[st];
      if (half == 0) {
        // thread = K position `row`: channel c, s1 and z in the record's builder order
        const int ch = dense_elem_of_kpos<BITS>(row), ka = kaux_of_elem(BITS, ch);
        const float s1 = e4m3_to_f32(kr[s1_off(BITS) + ka]);
        const float z = f16_bits_to_f32(reinterpret_cast<const uint16_t*>(kr + z_off(BITS))[ka]);
        reinterpret_cast<__half*>(sm.s1h)[row] = __float2half_rn(s1);                    // exact
        const float sz = s1 * z;
        const __half hi = __float2half_rn(sz), lo = __float2half_rn(sz - __half2float(hi));
        *reinterpret_cast<__half*>(sm.kt + kmaj_off(128, row, DN_KT)) = hi;
        *reinterpret_cast<__half*>(sm.kt + kmaj_off(129, row, DN_KT)) = lo;
      } else {
        // per-token aux of both records (parity-buffered: the softmax warps still read the previous chunk's)
        const float s1v = fmaxf(e4m3_to_f32(vr[s1_off(BITS) + slot_t]), 9.094947e-13f);
        const float zv = f16_bits_to_f32(reinterpret_cast<const uint16_t*>(vr + z_off(BITS))[slot_t]);
        sm.aux_a[st][rho_t] = make_float2(e4m3_to_f32(kr[s2_off(BITS) + slot_t]), lg2_approx(s1v));
        sm.aux_b[st][rho_t] = make_float2(rcp_approx(s1v), zv);
      }
      producer_sync();                                   // s1h complete
      {
        uint32_t W[2 * BITS];
        load_row_half<BITS>(kr, slot_t, half, W);
        dequant_half<BITS, true>(W, sm.s1h, __half2(), sm.kt, rho_t, DN_KT, half);
      }
      fence_async_smem();
      mbar_arrive(&sm.kt_full);
      producer_sync();                                   // every producer has left rec_k[st] and s1h
      if (pt == 0 && c + 2 < n_my) {
        mbar_expect_tx(&sm.full_k[st], RB); bulk_g2s(sm.rec_k[st], krec + (size_t)(c + 2) * RB, RB, &sm.full_k[st]);
      }
    };
    if (n_my > 0) expand_k(0);
    for (int it = 0; it < n_my; ++it) {
      const int st = it & 1;
      const uint32_t par = it & 1;
      if (it > 0) mbar_wait(&sm.bar_o[1], par ^ 1);      // PV of chunk it - 1 complete: Vt is free, softmax of it - 1 is over
      if (it + 1 < n_my) {                               // K of the NEXT chunk first: its QK^T overlaps this chunk's softmax
        mbar_wait(&sm.bar_s, par);                       // QK^T of this chunk has consumed Kt
        mbar_wait(&sm.s_free, par);                      // (*) the softmax warps have looked at kt_full of this chunk
        expand_k(it + 1);
      }
      mbar_wait(&sm.full_v[st], (it >> 1) & 1);
      {
        const uint8_t* vr = sm.rec_v[st];
        const float s2v = e4m3_to_f32(vr[s2_off(BITS) + row]);                           // thread = (channel row, token half)
        const __half2 sc = __float2half2_rn(s2v);
        uint32_t W[2 * BITS];
        load_row_half<BITS>(vr, row, half, W);
        dequant_half<BITS, false>(W, nullptr, sc, sm.vt, row, DN_KP, half);
        if (half == 0) *reinterpret_cast<__half2*>(sm.vt + kmaj_off(row, 128, DN_KP)) = sc;   // K columns 128, 129: s2v (zero-point term)
      }
      fence_async_smem();
      mbar_arrive(&sm.vt_full);
      producer_sync();                                   // every producer has left rec_v[st]
      if (pt == 0 && it + 2 < n_my) {
        mbar_expect_tx(&sm.full_v[st], RB); bulk_g2s(sm.rec_v[st], vrec + (size_t)(it + 2) * RB, RB, &sm.full_v[st]);
      }
    }
  } else if (warp == 16) {
    // =============================== MMA issuer: one thread =========================================================
    if (lane == 0) {
      auto issue_qk = [&](int c) {
        mbar_wait(&sm.kt_full, c & 1);
        if (c > 0) mbar_wait(&sm.s_free, (c & 1) ^ 1);    // the softmax warps have read S of the previous chunk
        tc_fence_after();
#pragma unroll
        for (int term = 0; term < 2; ++term)
#pragma unroll
          for (int ks = 0; ks < DN_KT / 16; ++ks)
            umma_f16(tmem, umma_desc(smem_u32(term ? sm.qlo : sm.qhi) + ks * 256, 128, SBO_T),
                     umma_desc(smem_u32(sm.kt) + ks * 256, 128, SBO_T), IDESC_S, (term | ks) != 0);
        umma_commit(&sm.bar_s);
      };
      if (n_my > 0) issue_qk(0);
      for (int it = 0; it < n_my; ++it) {
        const uint32_t par = it & 1;
        if (it + 1 < n_my) issue_qk(it + 1);              // runs while the softmax warps work on chunk it
        mbar_wait(&sm.vt_full, par);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          mbar_wait(&sm.p_full[h], par);
          tc_fence_after();
#pragma unroll
          for (int ks = 0; ks < DN_KPH / 16; ++ks) {      // 4 steps over the half's 64 tokens + 1 over the zero-point columns
            const uint32_t vcol = ks < 4 ? (uint32_t)(64 * h + 16 * ks) : 128u;
            umma_f16(tmem + O_COL + 128 * h, umma_desc(smem_u32(sm.pt[h]) + ks * 256, 128, SBO_PH),
                     umma_desc(smem_u32(sm.vt) + (vcol >> 3) * 128, 128, SBO_P), IDESC_O, (it | ks) != 0);
          }
          umma_commit(&sm.bar_o[h]);
        }
      }
    }
  } else {
    // =============================== softmax warps: thread = (query row = TMEM lane, token half) =====================
    const int h = warp >> 2, r = (warp & 3) * 32 + lane;
    const uint32_t t_row = tmem + ((uint32_t)((warp & 3) * 32) << 16);
    const uint32_t t_o = t_row + O_COL + 128 * h;
    uint8_t* prow = sm.pt[h] + (r >> 3) * SBO_PH + (r & 7) * 16;
    for (int it = 0; it < n_my; ++it) {
      const int st = it & 1;
      const uint32_t par = it & 1;
      mbar_wait(&sm.bar_s, par);
      mbar_wait(&sm.kt_full, par);                       // the producers' aux writes of this chunk are visible
      tc_fence_after();
      float v[64];
      float beta;
      {
        uint32_t b0, b1;
        tmem_ld2(t_row + 128, b0, b1);
        beta = __uint_as_float(b0) + __uint_as_float(b1);
        uint32_t u[16];
#pragma unroll
        for (int c0 = 0; c0 < 64; c0 += 16) {
          tmem_ld16(t_row + 64 * h + c0, u);
#pragma unroll
          for (int j = 0; j < 16; ++j) v[c0 + j] = __uint_as_float(u[j]);
        }
      }
      tc_fence_before();
      mbar_arrive(&sm.s_free);                           // S is in registers: the next QK^T may overwrite it
      const float2* aa = &sm.aux_a[st][64 * h];
      const float2* ab = &sm.aux_b[st][64 * h];
      float mx = -INFINITY;
#pragma unroll
      for (int j = 0; j < 64; ++j) {
        const float2 a = aa[j];
        v[j] = fmaf(a.x, v[j] + beta, a.y);
        mx = fmaxf(mx, v[j]);
      }
      const float m_new = fmaxf(m_ref, mx - P_OFF);
      const float f_old = ex2_approx(m_ref - m_new);     // 0 for the first chunk (m_ref = -inf)
      if (it > 0) {
        mbar_wait(&sm.bar_o[h], par ^ 1);                // PV of the previous chunk is complete: Pt is free, O is consistent
        tc_fence_after();
        if (__any_sync(0xffffffffu, m_new > m_ref)) {    // some row of the warp rises: rescale the accumulator rows in TMEM
#pragma unroll 1
          for (int c0 = 0; c0 < 128; c0 += 16) {
            uint32_t u[16];
            tmem_ld16(t_o + c0, u);
#pragma unroll
            for (int j = 0; j < 16; ++j) u[j] = __float_as_uint(__uint_as_float(u[j]) * f_old);
            tmem_st16(t_o + c0, u);
          }
          asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        }
      }
      m_ref = m_new;
      float lsum = 0.f, zsum = 0.f;
#pragma unroll
      for (int c0 = 0; c0 < 64; c0 += 8) {
        uint32_t o[4];
#pragma unroll
        for (int j = 0; j < 8; j += 2) {
          const float2 b0 = ab[c0 + j], b1 = ab[c0 + j + 1];
          const float p0 = ex2_approx(v[c0 + j] - m_new), p1 = ex2_approx(v[c0 + j + 1] - m_new);
          const __half2 ph = __floats2half2_rn(p0, p1);
          const float2 pf = __half22float2(ph);                 // the rounded values: numerator and denominator agree
          lsum = fmaf(pf.x, b0.x, fmaf(pf.y, b1.x, lsum));
          zsum = fmaf(pf.x, b0.y, fmaf(pf.y, b1.y, zsum));
          o[j >> 1] = *reinterpret_cast<const uint32_t*>(&ph);
        }
        *reinterpret_cast<uint4*>(prow + (c0 >> 3) * 128) = make_uint4(o[0], o[1], o[2], o[3]);
      }
      l_run = fmaf(l_run, f_old, lsum);
      {
        const __half zh = __float2half_rn(zsum), zl = __float2half_rn(zsum - __half2float(zh));
        *reinterpret_cast<__half2*>(prow + 8 * 128) = __halves2half2(zh, zl);              // K columns 64, 65
      }
      fence_async_smem();
      tc_fence_before();
      mbar_arrive(&sm.p_full[h]);
    }
  }
  // ---- epilogue, once per token half: O rows -> shared memory (the q tiles are dead: every QK^T has completed),
  //      inverse Hadamard, partial {m, l, o[128]} per query row into set DENSE_SETS * split + half ----------------------
  float* stage = reinterpret_cast<float*>(sm.qhi);       // [128][128] fp32 = qhi + qlo
#pragma unroll 1
  for (int hh = 0; hh < DENSE_SETS; ++hh) {
    if (warp < 8 && (warp >> 2) == hh) {
      const int r = (warp & 3) * 32 + lane;
      if (n_my > 0) {
        mbar_wait(&sm.bar_o[hh], (n_my - 1) & 1);
        tc_fence_after();
        const uint32_t t_o = tmem + ((uint32_t)((warp & 3) * 32) << 16) + O_COL + 128 * hh;
#pragma unroll 1
        for (int c0 = 0; c0 < 128; c0 += 16) {
          uint32_t u[16];
          tmem_ld16(t_o + c0, u);
#pragma unroll
          for (int j = 0; j < 16; j += 4)
            *reinterpret_cast<uint4*>(&stage[r * 128 + ((c0 + j) ^ ((r & 7) << 2))]) = make_uint4(u[j], u[j + 1], u[j + 2], u[j + 3]);
        }
      }
      sm.ml[r] = make_float2(m_ref, l_run);
      tc_fence_before();
    }
    __syncthreads();
    for (int r = warp; r < 128; r += DENSE_THREADS / 32) {
      const int R = rt * 128 + r;
      if (R >= n_rows) break;
      const int i = R / g, h = R - i * g;
      const size_t row = ((size_t)b * A.n_q + i) * A.Hq + hkv * g + h;
      float* prow = A.parts + ((size_t)(DENSE_SETS * split + hh) * ((size_t)A.B * A.n_q * A.Hq) + row) * PART_STRIDE;
      float v[4] = {0.f, 0.f, 0.f, 0.f};
      if (n_my > 0) {
        const float4 s4 = *reinterpret_cast<const float4*>(&stage[r * 128 + ((4 * lane) ^ ((r & 7) << 2))]);
        v[0] = s4.x; v[1] = s4.y; v[2] = s4.z; v[3] = s4.w;
        if (A.rotate_v) {
          fwht128_lane4(v, lane);
#pragma unroll
          for (int j = 0; j < 4; ++j) v[j] *= 0.08838834764831845f;
        }
      }
      *reinterpret_cast<float4*>(prow + 4 + 4 * lane) = make_float4(v[0], v[1], v[2], v[3]);
      if (lane == 0) {
        const float2 ml = sm.ml[r];
        *reinterpret_cast<float4*>(prow) = make_float4(n_my > 0 ? ml.x : -INFINITY, n_my > 0 ? ml.y : 0.f, 0.f, 0.f);
      }
    }
    __syncthreads();
  }
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(TMEM_COLS));
}

}  // namespace kvarn

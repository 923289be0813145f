// Dense multi-token read path on the 5th-generation tensor cores (tcgen05 + TMEM): a block of query rows against the
// packed chunks of the cache (Fig. 4 pseudo-decode).  Used by kvarn_block_attention_dense
// for blocks with many (query token, head) rows per KV head.  The raw windows (sink, residual, the block's own causal
// tokens) run through the same pipeline as extra chunks after the packed ones (rotated rows as fp16 tiles, K in two
// terms, masked in the softmax); the partial sets of all CTAs are merged by merge_partials_kernel.
//
// One CTA = one (sequence, KV head), one tile of 128 query rows r = (token i, head h), one range of chunks; three roles
// that meet only through mbarriers: warps 8-15 expand the records (producers), one thread of warp 16 issues the MMAs,
// warps 0-7 own the softmax (thread = (query row = TMEM lane, token half)).  Per chunk:
//   K record --TMA--> shared memory --producers--> Kt = code x s1[c] as fp16 (EXACT: a 2-/4-bit code times an E4M3
//     scale has <= 8 significant bits), K-major UMMA tile [token][channel], + two rows hi / lo of (s1 z)[c] for beta
//   S[r][t] = sum_c (q'_hi + q'_lo)[r][c] Kt[t][c]          tcgen05.mma kind::f16, M = 128, N = 144, K = 128, twice (hi, lo)
//   logit = s2[t] (S + beta_r) + E;  online softmax per (row, token half) inside one thread; the two halves are
//     independent streams (own reference exponent, l, accumulator) and leave two partial sets
//   p~ = 2^(logit - m + 8) as fp16 pairs, written to tensor memory (+ hi / lo of the zero-point sum as two extra K columns)
//   V record --> Vt = (codeV x s2v[c]) x f_t as fp16 (exact; f_t = s1v[t] 2^-E, E = largest s1v exponent of the chunk),
//     [channel][token] (+ s2v[c] in the extra K columns)
//   O_h[r][c] += sum_t p~[r][t] Vt[c][t]                    tcgen05.mma, A from tensor memory, M = 128, N = 128, K = 80
// The accumulators are rescaled in TMEM (tcgen05.ld / st) only when a row's maximum rises.  Finally each O_h is
// un-rotated (inverse Hadamard) and written as the partial {m, l, o[128]} of its rows.  While the softmax warps work on
// chunk i the producers expand K of chunk i + 1 (second Kt buffer) and V of chunk i, and QK^T of chunk i + 1 runs.
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
  const void* k_resid; const void* v_resid;   // raw residual window [B * Hkv][128][128]
  const void* k_sink;  const void* v_sink;    // raw sink tokens [B * Hkv][n_sink][128]
  const void* k_blk;   const void* v_blk;     // the block's own tokens [B * Hkv][n_q][128] (causal), or null
  float* parts;         // [splits][B * n_q * Hq][PART_STRIDE] (splits > 1)
  void* out;            // splits == 1: the normalised result [B][n_q][Hq][128] is written directly
  int out_dtype;
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
// A operand from tensor memory (lane = row, one 32-bit column = two consecutive K elements)
__device__ __forceinline__ void umma_f16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
               ::"r"(d_tmem), "r"(a_tmem), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
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
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t (&v)[8]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
               ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]) : "memory");
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

// Kt and Vt are written by the producers with 16-byte stores from lanes that hold different 8-column units of
// different rows.  Their core matrices are therefore spread with LBO = 144 B (K direction) and an odd number of
// 16-byte groups per 8 rows (SBO): with the lane assignment of ProducerLane every quarter warp then stores to eight
// different bank groups, and its record loads are one contiguous 128 B line per warp (no bank conflict on either side).
constexpr int DN_NO_MASK = 1 << 20;
constexpr int DN_LBO = 144;
constexpr int DN_SBO_K = (16 * 9 + 1) * 16;      // 2320 B per 8 rows of Kt (16 units of 144 B + 16 B)
constexpr int DN_SBO_V = (18 * 9 + 1) * 16;      // 2608 B per 8 rows of Vt (18 units + 16 B)
__host__ __device__ constexpr int tile_off(int r, int k, int SBO) {
  return (r >> 3) * SBO + (k >> 3) * DN_LBO + (r & 7) * 16 + (k & 7) * 2;
}

// inverse of slot_of_token
__host__ __device__ constexpr int token_of_slot(int bits, int s) {
  return bits == 2 ? (((s >> 5) & 3) | (((s >> 3) & 1) << 2) | (((s >> 4) & 1) << 3) | ((s & 3) << 4) | (((s >> 2) & 1) << 6))
                   : (((s >> 5) & 1) | (((s >> 3) & 1) << 1) | (((s >> 4) & 1) << 2) | ((s & 3) << 3) | (((s >> 2) & 1) << 5) |
                      (((s >> 6) & 1) << 6));
}
constexpr bool token_slot_roundtrip(int bits) {
  for (int t = 0; t < 128; ++t)
    if (token_of_slot(bits, slot_of_token(bits, t)) != t) return false;
  return true;
}
static_assert(token_slot_roundtrip(2) && token_slot_roundtrip(4), "token_of_slot must invert slot_of_token");

template <int BITS>
struct DenseSmem {
  static constexpr int RB = record_bytes(BITS);
  alignas(1024) uint8_t qhi[128 * DN_KT * 2];      // q' (rotated, scaled), first fp16 term; later: staging of O (with qlo)
  alignas(1024) uint8_t qlo[128 * DN_KT * 2];      // second fp16 term
  alignas(128) uint8_t kt[2][18 * DN_SBO_K];       // [chunk parity] rows 0..127: token rho(t); 128, 129: hi / lo of s1 z; 130..143: zero
  alignas(128) uint8_t vt[16 * DN_SBO_V];          // rows: channels; columns 0..127 tokens (rho order), 128, 129: s2v, rest zero
  alignas(128) uint8_t rec_k[2][RB];               // [chunk parity]
  alignas(128) uint8_t rec_v[2][RB - 512];         // the codes of the V record
  alignas(128) uint8_t aux_v[3][512];              // [chunk % 3] its s1 | s2 | z (requested two chunks earlier than the codes)
  alignas(16) __half2 s1h[64];                     // s1 of the K record as fp16 pairs in K-position order
  alignas(16) __half2 s1n[64];                     // the addends -dq_bias s1 of the same pairs
  alignas(16) __half2 fh[2][64];                   // [chunk parity] f_t = s1v[t] 2^-E of the V record, pairs in K-position order
  alignas(16) float2 aux_s2[3][64];                // [chunk % 3] per token pair (rho order): s2 of the K record
  alignas(16) float2 aux_zm[3][64];                //                                         f_t zv[t] of the V record
  alignas(8) float2 e_chunk[3];                    // [chunk % 3] {E, 2^-E}: E = largest binary exponent of the chunk's s1v
  alignas(8) int2 mask[3];                         // [chunk % 3] {tokens in the chunk, vis0}: column n is visible to query token i
                                                   // iff n < tokens and n <= vis0 + i (raw chunks; packed: {128, DN_NO_MASK})
  int e_warp[4];
  __device__ float2* ml() { return reinterpret_cast<float2*>(rec_k[0]); }   // epilogue: {m, l} of the rows (records are dead)
  alignas(8) uint64_t full_k[2], full_v[2];        // TMA arrival [chunk parity]
  alignas(8) uint64_t full_va[3];                  // TMA arrival of aux_v [chunk % 3]
  alignas(8) uint64_t bar_s, bar_o[2];             // MMA completion (tcgen05.commit): S ready, O of a token half accumulated
  alignas(8) uint64_t kt_full[2], vt_full;         // producers -> issuer, one arrival per warp
  alignas(8) uint64_t aux_full[3];                 // producers -> softmax warps: aux of chunk c in slot c % 3
  alignas(8) uint64_t k_free[2];                   // tcgen05.commit: the QK^T that read kt[parity] has completed
  alignas(8) uint64_t s_free, p_full[2];           // softmax warps -> issuer (256 / 128 arrivals)
  uint32_t tmem_base;
};

// Producer thread (warp pw = 0..7, lane): pw = (w, mtile) of the record's slot numbering; the lane names
// (g & 1, t, rho, word quarter) so that iteration i of a warp reads the 128 contiguous bytes
// [w, mtile(, rho)] + 128 i of the code block.  The thread's word index `wi` is the same in every iteration: its
// scales live in registers for the whole chunk.
template <int BITS>
struct ProducerLane {
  int glo, t, rho, q;      // 2-bit: q = which half of the 8 words; 4-bit: q = which quarter of the 16 words, rho unused
  __device__ __forceinline__ explicit ProducerLane(int lane) {
    glo = lane >> 4; t = (lane >> 1) & 3;
    if constexpr (BITS == 2) { rho = lane & 1; q = (lane >> 3) & 1; }
    else { rho = 0; q = (lane & 1) | (((lane >> 3) & 1) << 1); }
  }
  __device__ __forceinline__ int wi() const { return 4 * q + t; }
  static constexpr int ITERS = BITS == 2 ? 4 : 8;
  // byte offset of the word inside the code block, slot of its row
  __device__ __forceinline__ int word_off(int pw, int it) const {
    const int w = pw >> 1, mt = pw & 1;
    if constexpr (BITS == 2) return w * 1024 + mt * 512 + it * 128 + glo * 64 + t * 16 + rho * 8 + q * 4;
    else return w * 2048 + mt * 1024 + (it >> 2) * 512 + (it & 3) * 128 + glo * 64 + t * 16 + q * 4;
  }
  __device__ __forceinline__ int slot(int pw, int it) const {
    const int w = pw >> 1, mt = pw & 1;
    if constexpr (BITS == 2) return w * 32 + mt * 16 + rho * 8 + 2 * it + glo;
    else return w * 32 + mt * 16 + (it >> 2) * 8 + 2 * (it & 3) + glo;
  }
};

// Expansion of a code pair without un-biasing: the two codes of pair j of a word (codes j and j + CPW / 2) are moved to
// mantissa bits [p, p + BITS) of the two fp16 lanes, p = dq_p(j) >= 4, under the exponent of 2^(10 - p): the lanes then
// hold 2^(10 - p) + code, and ONE fma gives code * s = (2^(10 - p) + code) * s - 2^(10 - p) s, exactly (the product is
// exact inside the fma, the result has <= 8 significant bits, the addend is at most 64 * 448).  Three (2-bit) codes
// share one shifted copy of the word.
template <int BITS> __host__ __device__ constexpr int dq_p(int j) { return BITS == 2 ? 4 + 2 * (j % 3) : 4; }
template <int BITS> __host__ __device__ constexpr float dq_bias(int j) { return (float)(1 << (10 - dq_p<BITS>(j))); }

// One packed word (CPW codes = CPW consecutive K positions) of a row -> fp16 values, written as CPW / 8 units of
// 16 bytes at `dst` (+ DN_LBO per unit).  K: value = code * s[j] via add[j] = -dq_bias s[j].  V: value =
// (code * sc) * f[j]: both products exact (<= 8, then <= 11 significant bits).
template <int BITS, bool IS_K>
__device__ __forceinline__ void dequant_word(uint32_t W, const __half2 (&s)[16 / BITS], const __half2 (&add)[16 / BITS],
                                             __half2 sc, const __half2 (&nsc)[3], uint8_t* dst) {
  constexpr int PPW = 16 / BITS;
  constexpr uint32_t MASK = BITS == 2 ? 0x00030003u : 0x000F000Fu;
  uint32_t o[PPW];
#pragma unroll
  for (int j = 0; j < PPW; ++j) {
    const int p = dq_p<BITS>(j), delta = p - BITS * j;
    const uint32_t Wg = delta >= 0 ? (W << delta) : (W >> (-delta));
    uint32_t h = (Wg & (MASK << p)) | (((uint32_t)(25 - p) << 10) * 0x00010001u);
    __half2 x;
    if constexpr (IS_K) x = __hfma2(*reinterpret_cast<__half2*>(&h), s[j], add[j]);
    else x = __hmul2(__hfma2(*reinterpret_cast<__half2*>(&h), sc, nsc[BITS == 2 ? j % 3 : 0]), s[j]);
    o[j] = *reinterpret_cast<uint32_t*>(&x);
  }
#pragma unroll
  for (int u = 0; u < PPW / 4; ++u)
    *reinterpret_cast<uint4*>(dst + u * DN_LBO) = make_uint4(o[4 * u], o[4 * u + 1], o[4 * u + 2], o[4 * u + 3]);
}

__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// one arrival per warp: the lanes' writes are ordered before it by the warp barrier
__device__ __forceinline__ void mbar_arrive_warp(uint64_t* bar, int lane) {
  __syncwarp();
  if (lane == 0) mbar_arrive(bar);
}
__device__ __forceinline__ void producer_sync() { asm volatile("bar.sync 1, 256;" ::: "memory"); }
__device__ __forceinline__ void tmem_ld2(uint32_t taddr, uint32_t& a, uint32_t& b) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0,%1}, [%2];" : "=r"(a), "=r"(b) : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}




static_assert(sizeof(DenseSmem<2>) <= 231424 && sizeof(DenseSmem<4>) <= 231424, "dense tiles exceed the shared memory of one SM");
constexpr int DENSE_THREADS = 640;          // warps 0-7 softmax, 8-15 producers, 16 MMA issuer (17-19 idle: whole warpgroups
                                            // for setmaxnreg)
// 96 registers per thread at launch (640 threads), re-divided: the softmax warps keep 64 logits plus prefetched aux live
constexpr int DENSE_REGS_SOFTMAX = 120, DENSE_REGS_PRODUCER = 72;
template <int N> __device__ __forceinline__ void setmaxnreg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void setmaxnreg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
__device__ __forceinline__ void softmax_sync() { asm volatile("bar.sync 2, 256;" ::: "memory"); }
constexpr int DENSE_SETS = 1;               // partial sets per CTA (the two token-half streams are merged in the epilogue)

template <int BITS, typename InT>
__global__ void __launch_bounds__(DENSE_THREADS, 1) block_dense_kernel(const DenseArgs A) {
  using SM = DenseSmem<BITS>;
  constexpr int RB = SM::RB;
  constexpr int PPW = 16 / BITS, CPW = 32 / BITS;
  // tensor memory: S: columns [0, 144); p~ of token half h (fp16 pairs, the A operand of PV): [144 + 40 h, 184 + 40 h);
  // O of token half h: [256 + 128 h, 384 + 128 h)
  constexpr uint32_t TMEM_COLS = 512;
  constexpr uint32_t P_COL = 144, O_COL = 256;
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
  // Raw windows run through the same pipeline as extra chunks after the packed ones: their K / V rows are rotated and
  // rounded to fp16 by the producers (one term: 2^-12 per element, below the other terms of the tolerance), s2 = 1, no
  // zero point, and the softmax masks by count and causality.  Sink: split 0; residual window and the block's own
  // tokens: the last split.
  const InT* raw_k[3]; const InT* raw_v[3]; int raw_cnt[3], raw_vis[3];
  int n_raw = 0;
  {
    const int ns_tok = min(len, A.n_sink), resid = body & 127;
    if (split == 0 && ns_tok > 0) {
      raw_k[n_raw] = reinterpret_cast<const InT*>(A.k_sink) + (size_t)unit * A.n_sink * D;
      raw_v[n_raw] = reinterpret_cast<const InT*>(A.v_sink) + (size_t)unit * A.n_sink * D;
      raw_cnt[n_raw] = ns_tok; raw_vis[n_raw] = DN_NO_MASK; ++n_raw;
    }
    if (split == A.splits - 1 && resid > 0) {
      raw_k[n_raw] = reinterpret_cast<const InT*>(A.k_resid) + (size_t)unit * G * D;
      raw_v[n_raw] = reinterpret_cast<const InT*>(A.v_resid) + (size_t)unit * G * D;
      raw_cnt[n_raw] = resid; raw_vis[n_raw] = DN_NO_MASK; ++n_raw;
    }
    if (split == A.splits - 1 && A.k_blk != nullptr) {
      raw_k[n_raw] = reinterpret_cast<const InT*>(A.k_blk) + (size_t)unit * A.n_q * D;
      raw_v[n_raw] = reinterpret_cast<const InT*>(A.v_blk) + (size_t)unit * A.n_q * D;
      raw_cnt[n_raw] = A.n_q; raw_vis[n_raw] = 0; ++n_raw;
    }
  }
  const int n_tot = n_my + n_raw;
  const int n_rows = A.n_q * g;                                                     // query rows of this (b, kv head)
  const uint8_t* krec = A.k_records + ((size_t)unit * A.max_chunks + c_begin) * RB;
  const uint8_t* vrec = A.v_records + ((size_t)unit * A.max_chunks + c_begin) * RB;

  // ---- setup: barriers, TMEM, first records, q ------------------------------------------------------------------
  if (tid == 256) {
    for (int s = 0; s < 2; ++s) { mbar_init(&sm.full_k[s], 1); mbar_init(&sm.full_v[s], 1); mbar_init(&sm.bar_o[s], 1); mbar_init(&sm.p_full[s], 4);
                                  mbar_init(&sm.kt_full[s], 8); mbar_init(&sm.k_free[s], 1); }
    for (int s = 0; s < 3; ++s) { mbar_init(&sm.full_va[s], 1); mbar_init(&sm.aux_full[s], 8); }
    mbar_init(&sm.bar_s, 1);
    mbar_init(&sm.vt_full, 8); mbar_init(&sm.s_free, 8);                                 // one arrival per warp
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    for (int c = 0; c < 2 && c < n_my; ++c) {
      mbar_expect_tx(&sm.full_k[c], RB); bulk_g2s(sm.rec_k[c], krec + (size_t)c * RB, RB, &sm.full_k[c]);
      mbar_expect_tx(&sm.full_v[c], RB - 512); bulk_g2s(sm.rec_v[c], vrec + (size_t)c * RB, RB - 512, &sm.full_v[c]);
    }
    for (int c = 0; c < 3 && c < n_my; ++c) {
      mbar_expect_tx(&sm.full_va[c], 512); bulk_g2s(sm.aux_v[c], vrec + (size_t)c * RB + (RB - 512), 512, &sm.full_va[c]);
    }
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&sm.tmem_base)), "n"(TMEM_COLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  // q' = (q H / sqrt(128)) q_scale as two fp16 terms, columns in K-position order.  Two steps, so that both sides of shared
  // memory are conflict-free: (1) a warp rotates a row (lane = 4 channels) and writes it as fp32 into a scratch
  // [128][132] that borrows the Kt buffers; (2) lane = (row of an 8-row group, unit of 8 K positions) reads its eight values
  // and stores them as one 16-byte piece of the hi and of the lo tile: a quarter warp covers 128 contiguous bytes.
  // (Writing 2-byte pieces straight from step 1 cost 16-way conflicts: 10 us per CTA.)
  constexpr int QS = 132;                                                        // scratch row stride in floats
  float* qscr = reinterpret_cast<float*>(sm.kt);
  static_assert(sizeof(sm.kt) >= 128 * QS * sizeof(float), "q scratch borrows the Kt buffers");
  constexpr int QROWS = (128 + DENSE_THREADS / 32 - 1) / (DENSE_THREADS / 32);   // rows per warp: all loads in flight together
  float qv[QROWS][4];
#pragma unroll
  for (int k = 0; k < QROWS; ++k) {
    const int r = warp + k * (DENSE_THREADS / 32), R = rt * 128 + r;
#pragma unroll
    for (int j = 0; j < 4; ++j) qv[k][j] = 0.f;
    if (r < 128 && R < n_rows) {
      const int i = R / g, h = R - i * g;
      const size_t row = ((size_t)b * A.n_q + i) * A.Hq + hkv * g + h;
      const InT* qp = reinterpret_cast<const InT*>(A.q) + row * D + 4 * lane;
#pragma unroll
      for (int j = 0; j < 4; ++j) qv[k][j] = ld_in<InT>(qp + j) * A.q_scale;
    }
  }
#pragma unroll
  for (int k = 0; k < QROWS; ++k) {
    const int r = warp + k * (DENSE_THREADS / 32);
    if (r >= 128) break;
    float v[4] = {qv[k][0], qv[k][1], qv[k][2], qv[k][3]};
    if (A.rotate_k) {
      fwht128_lane4(v, lane);
#pragma unroll
      for (int j = 0; j < 4; ++j) v[j] *= 0.08838834764831845f;
    }
    *reinterpret_cast<float4*>(&qscr[r * QS + 4 * lane]) = make_float4(v[0], v[1], v[2], v[3]);
  }
  __syncthreads();
  for (int w = warp; w < 16 * 4; w += DENSE_THREADS / 32) {                      // (row group, quarter of the 16 units)
    const int r = (w >> 2) * 8 + (lane & 7), u = (w & 3) * 4 + (lane >> 3);
    const int e0 = dense_elem_of_kpos<BITS>(8 * u), e1 = dense_elem_of_kpos<BITS>(8 * u + 1);   // K positions 8u + 2i / + 2i + 1 = elements e0 + i / e1 + i
    const float4 a = *reinterpret_cast<const float4*>(&qscr[r * QS + e0]);
    const float4 c = *reinterpret_cast<const float4*>(&qscr[r * QS + e1]);
    const float x[8] = {a.x, c.x, a.y, c.y, a.z, c.z, a.w, c.w};
    uint32_t hi[4], lo[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const __half2 h2 = __floats2half2_rn(x[2 * i], x[2 * i + 1]);
      const float2 hf = __half22float2(h2);
      const __half2 l2 = __floats2half2_rn(x[2 * i] - hf.x, x[2 * i + 1] - hf.y);
      hi[i] = *reinterpret_cast<const uint32_t*>(&h2); lo[i] = *reinterpret_cast<const uint32_t*>(&l2);
    }
    *reinterpret_cast<uint4*>(sm.qhi + kmaj_off(r, 8 * u, DN_KT)) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
    *reinterpret_cast<uint4*>(sm.qlo + kmaj_off(r, 8 * u, DN_KT)) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
  }
  __syncthreads();
  // zero the tiles once: rows / columns that are never rewritten (padding of N = 144 and of the K extents) stay zero
  for (int i = tid; i < (int)(sizeof(sm.kt) / 16); i += DENSE_THREADS) reinterpret_cast<uint4*>(sm.kt)[i] = make_uint4(0, 0, 0, 0);
  for (int i = tid; i < (int)(sizeof(sm.vt) / 16); i += DENSE_THREADS) reinterpret_cast<uint4*>(sm.vt)[i] = make_uint4(0, 0, 0, 0);
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = sm.tmem_base;
  constexpr uint32_t IDESC_S = umma_idesc_f16(128, DN_NS), IDESC_O = umma_idesc_f16(128, 128);
  constexpr uint32_t SBO_T = (DN_KT / 8) * 128;
  constexpr float P_OFF = 8.f;                  // p~ = 2^(logit - max + 8): probabilities down to 2^-32 of the maximum survive fp16
  float m_ref = -INFINITY, l_run = 0.f;         // softmax warps: reference exponent of the (row, token half), running l

  // Barrier phases: phase i of kt_full / vt_full / s_free / p_full / bar_s / bar_o belongs to chunk i (parity i & 1).  No
  // barrier completes phase i + 1 before every waiter of phase i has looked (a parity wait cannot tell i from i + 2):
  // the waits marked (*) below are there for that reason alone.
  if (warp >= 8 && warp < 16) {
    // =============================== producers ======================================================================
    setmaxnreg_dec<DENSE_REGS_PRODUCER>();
    const int pt = tid - 256, pw = warp - 8;
    const ProducerLane<BITS> L(lane);
    const int wi = L.wi();
    // per-thread constants of the aux phase: threads 0..127 own S column / K position n = pt of the token axis,
    // threads 128..255 own K position pt - 128 of the channel axis
    const int n_ax = pt & 127;
    const int tok = dense_elem_of_kpos<BITS>(n_ax), slot_tok = slot_of_token(BITS, tok);
    const int ka = kaux_of_elem(BITS, dense_elem_of_kpos<BITS>(n_ax));
    // tile rows of the thread's words: Kt row = S column of the slot's token, Vt row = slot (channel)
    int krow_off[ProducerLane<BITS>::ITERS], vrow_off[ProducerLane<BITS>::ITERS];
#pragma unroll
    for (int i = 0; i < ProducerLane<BITS>::ITERS; ++i) {
      const int sl = L.slot(pw, i);
      const int kr_ = dense_kpos<BITS>(token_of_slot(BITS, sl));
      krow_off[i] = tile_off(kr_, 0, DN_SBO_K) + wi * (CPW / 8) * DN_LBO;
      vrow_off[i] = tile_off(sl, 0, DN_SBO_V) + wi * (CPW / 8) * DN_LBO;
    }
    // rows pw, pw + 8, ... < cnt of a raw window, rotated, four rows' loads in flight together
    auto raw_rows = [&](const InT* base, int cnt, int rotate, auto store) {
      for (int t0 = pw; t0 < cnt; t0 += 32) {
        float x[4][4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const int t = t0 + 8 * k;
#pragma unroll
          for (int e = 0; e < 4; ++e) x[k][e] = t < cnt ? ld_in<InT>(base + (size_t)t * D + 4 * lane + e) : 0.f;
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const int t = t0 + 8 * k;
          if (t >= cnt) break;
          if (rotate) {
            fwht128_lane4(x[k], lane);
#pragma unroll
            for (int e = 0; e < 4; ++e) x[k][e] *= 0.08838834764831845f;
          }
          store(t, x[k]);
        }
      }
    };
    // chunk c: aux of both records, then Kt; afterwards the K record of chunk c + 2 is requested
    auto expand_k = [&](int c) {
      const int st = c & 1, s3 = c % 3;
      const uint32_t par_rec = (c >> 1) & 1;
      if (c >= n_my) {
        // raw chunk: Kt row n = token n (identity order), columns in the K-position order of q'
        // The rotated row enters as TWO fp16 terms (keys have outlier channels of several hundred: one term would cost
        // 1e-2 of a logit): the first in kt[st], the second in the Vt buffer laid out as a 128-row K tile -- which is why
        // raw chunks are not prefetched: Vt is free only when PV of the previous chunk has completed.
        const int j = c - n_my;
        if (c >= 2) mbar_wait(&sm.k_free[st], par_rec ^ 1);
        if (c >= 1) mbar_wait(&sm.bar_o[1], (c & 1) ^ 1);
        uint8_t* kt = sm.kt[st];
        if (pt < 128) {
          reinterpret_cast<float*>(&sm.aux_s2[s3][n_ax >> 1])[n_ax & 1] = 1.f;
          reinterpret_cast<float*>(&sm.aux_zm[s3][n_ax >> 1])[n_ax & 1] = 0.f;
          if (pt == 0) { sm.e_chunk[s3] = make_float2(0.f, 1.f); sm.mask[s3] = make_int2(raw_cnt[j], raw_vis[j]); }
        } else {
          *reinterpret_cast<__half*>(kt + tile_off(128, n_ax, DN_SBO_K)) = __float2half_rn(0.f);   // no beta
          *reinterpret_cast<__half*>(kt + tile_off(129, n_ax, DN_SBO_K)) = __float2half_rn(0.f);
        }
        const InT* kp = raw_k[j];
        const int cnt = raw_cnt[j];
        // only the rows of real tokens: rows >= cnt keep stale (finite) tile contents and are masked in the softmax
        raw_rows(kp, cnt, A.rotate_k, [&](int t, const float (&x)[4]) {
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const int off = tile_off(t, dense_kpos<BITS>(4 * lane + e), DN_SBO_K);
            const __half hi = __float2half_rn(x[e]);
            *reinterpret_cast<__half*>(kt + off) = hi;
            *reinterpret_cast<__half*>(sm.vt + off) = __float2half_rn(x[e] - __half2float(hi));
          }
        });
        fence_async_smem();
        __syncwarp();
        if (lane == 0) { mbar_arrive(&sm.kt_full[st]); mbar_arrive(&sm.aux_full[s3]); }
        producer_sync();
        return;
      }
      mbar_wait(&sm.full_k[st], par_rec);
      mbar_wait(&sm.full_va[s3], (c / 3) & 1);
      if (c >= 2) mbar_wait(&sm.k_free[st], par_rec ^ 1);  // the QK^T of chunk c - 2 has consumed kt[st]
      const uint8_t* kr = sm.rec_k[st];
      const uint8_t* va = sm.aux_v[s3];                    // s1 at 0, s2 at 128, z at 256
      uint8_t* kt = sm.kt[st];
      float s1v = 0.f;
      if (pt < 128) {
        // binary exponent of s1v[token]; E = the largest of the chunk (through e_warp)
        s1v = e4m3_to_f32(va[slot_tok]);
        const int e = s1v > 0.f ? (int)((__float_as_uint(s1v) >> 23) & 0xFF) - 127 : -64;
        const int em = __reduce_max_sync(0xffffffffu, e);
        if (lane == 0) sm.e_warp[pw] = em;
      } else {
        // channel of K position n_ax: s1 and z in the record's builder order
        const float s1 = e4m3_to_f32(kr[s1_off(BITS) + ka]);
        const float z = f16_bits_to_f32(reinterpret_cast<const uint16_t*>(kr + z_off(BITS))[ka]);
        reinterpret_cast<__half*>(sm.s1h)[n_ax] = __float2half_rn(s1);                    // exact
        reinterpret_cast<__half*>(sm.s1n)[n_ax] = __float2half_rn(-dq_bias<BITS>((n_ax >> 1) % PPW) * s1);
        const float sz = s1 * z;
        const __half hi = __float2half_rn(sz), lo = __float2half_rn(sz - __half2float(hi));
        *reinterpret_cast<__half*>(kt + tile_off(128, n_ax, DN_SBO_K)) = hi;
        *reinterpret_cast<__half*>(kt + tile_off(129, n_ax, DN_SBO_K)) = lo;
      }
      producer_sync();                                   // s1h, s1n, e_warp complete
      if (pt < 128) {
        const int E = max(max(sm.e_warp[0], sm.e_warp[1]), max(sm.e_warp[2], sm.e_warp[3]));
        const float two_mE = __uint_as_float((uint32_t)(127 - max(E, -64)) << 23);        // 2^-E
        const float f = s1v * two_mE;                    // in [0, 2): the V tile carries s2v f, the logits carry E
        const float zv = f16_bits_to_f32(reinterpret_cast<const uint16_t*>(va + 256)[slot_tok]);
        reinterpret_cast<__half*>(sm.fh[st])[n_ax] = __float2half_rn(f);
        reinterpret_cast<float*>(&sm.aux_s2[s3][n_ax >> 1])[n_ax & 1] = e4m3_to_f32(kr[s2_off(BITS) + slot_tok]);
        reinterpret_cast<float*>(&sm.aux_zm[s3][n_ax >> 1])[n_ax & 1] = f * zv;
        if (pt == 0) { sm.e_chunk[s3] = make_float2((float)max(E, -64), two_mE); sm.mask[s3] = make_int2(128, DN_NO_MASK); }
      }
      {
        __half2 sK[PPW], aK[PPW];
        const __half2 nsc0[3] = {__half2(), __half2(), __half2()};
#pragma unroll
        for (int j = 0; j < PPW; j += 4) {
          const uint4 s4 = *reinterpret_cast<const uint4*>(&sm.s1h[wi * PPW + j]);
          const uint4 a4 = *reinterpret_cast<const uint4*>(&sm.s1n[wi * PPW + j]);
          sK[j] = *reinterpret_cast<const __half2*>(&s4.x); sK[j + 1] = *reinterpret_cast<const __half2*>(&s4.y);
          sK[j + 2] = *reinterpret_cast<const __half2*>(&s4.z); sK[j + 3] = *reinterpret_cast<const __half2*>(&s4.w);
          aK[j] = *reinterpret_cast<const __half2*>(&a4.x); aK[j + 1] = *reinterpret_cast<const __half2*>(&a4.y);
          aK[j + 2] = *reinterpret_cast<const __half2*>(&a4.z); aK[j + 3] = *reinterpret_cast<const __half2*>(&a4.w);
        }
        uint32_t W[ProducerLane<BITS>::ITERS];
#pragma unroll
        for (int i = 0; i < ProducerLane<BITS>::ITERS; ++i) W[i] = *reinterpret_cast<const uint32_t*>(kr + L.word_off(pw, i));
#pragma unroll
        for (int i = 0; i < ProducerLane<BITS>::ITERS; ++i)
          dequant_word<BITS, true>(W[i], sK, aK, __half2(), nsc0, kt + krow_off[i]);
      }
      fence_async_smem();
      __syncwarp();
      if (lane == 0) { mbar_arrive(&sm.kt_full[st]); mbar_arrive(&sm.aux_full[s3]); }
      producer_sync();                                   // every producer has left rec_k[st], s1h, s1n, e_warp
      if (pt == 0 && c + 2 < n_my) {
        mbar_expect_tx(&sm.full_k[st], RB); bulk_g2s(sm.rec_k[st], krec + (size_t)(c + 2) * RB, RB, &sm.full_k[st]);
      }
    };
    if (n_my > 0) expand_k(0);
    for (int it = 0; it < n_tot; ++it) {
      const int st = it & 1;
      const uint32_t par = it & 1;
      if (it >= n_my) expand_k(it);                      // raw chunk: expanded in its own turn (it waits for PV of chunk it - 1)
      else if (it + 1 < n_my) expand_k(it + 1);          // K of the NEXT chunk first: its QK^T overlaps this chunk's softmax
      if (it < n_my) {
        mbar_wait(&sm.full_v[st], (it >> 1) & 1);
        if (it > 0) mbar_wait(&sm.bar_o[1], par ^ 1);    // PV of chunk it - 1 complete: Vt is free, softmax of it - 1 is over
      } else {
        mbar_wait(&sm.bar_s, par);                       // QK^T of this chunk has consumed the second K term in the Vt buffer
      }
      if (it >= n_my) {
        // raw chunk: Vt[channel][token n] = fp16 of the rotated V row n
        const int j = it - n_my;
        const InT* vp = raw_v[j];
        const int cnt = raw_cnt[j];
        // (columns >= cnt keep stale finite values: their p~ is exactly zero)
        raw_rows(vp, cnt, A.rotate_v, [&](int t, const float (&x)[4]) {
#pragma unroll
          for (int e = 0; e < 4; ++e)
            *reinterpret_cast<__half*>(sm.vt + tile_off(4 * lane + e, t, DN_SBO_V)) = __float2half_rn(x[e]);
        });
      } else {
        uint8_t* vt = sm.vt;
        const uint8_t* vr = sm.rec_v[st];
        const uint8_t* va = sm.aux_v[it % 3];
        __half2 fV[PPW];
#pragma unroll
        for (int j = 0; j < PPW; j += 4) {
          const uint4 f4 = *reinterpret_cast<const uint4*>(&sm.fh[st][wi * PPW + j]);
          fV[j] = *reinterpret_cast<const __half2*>(&f4.x); fV[j + 1] = *reinterpret_cast<const __half2*>(&f4.y);
          fV[j + 2] = *reinterpret_cast<const __half2*>(&f4.z); fV[j + 3] = *reinterpret_cast<const __half2*>(&f4.w);
        }
        uint32_t W[ProducerLane<BITS>::ITERS];
#pragma unroll
        for (int i = 0; i < ProducerLane<BITS>::ITERS; ++i) W[i] = *reinterpret_cast<const uint32_t*>(vr + L.word_off(pw, i));
#pragma unroll
        for (int i = 0; i < ProducerLane<BITS>::ITERS; ++i) {
          const __half2 sc = __float2half2_rn(e4m3_to_f32(va[128 + L.slot(pw, i)]));   // s2v of the row's channel
          __half2 nsc[3];
#pragma unroll
          for (int k = 0; k < 3; ++k) nsc[k] = __hmul2(sc, __float2half2_rn(-dq_bias<BITS>(k)));
          dequant_word<BITS, false>(W[i], fV, fV, sc, nsc, vt + vrow_off[i]);
        }
        if (pt < 128)                                    // K columns 128, 129 of channel row pt: s2v (zero-point term)
          *reinterpret_cast<__half2*>(vt + tile_off(pt, 128, DN_SBO_V)) = __float2half2_rn(e4m3_to_f32(va[128 + pt]));
      }
      fence_async_smem();
      mbar_arrive_warp(&sm.vt_full, lane);
      producer_sync();                                   // every producer has left rec_v[st] and aux_v[it % 3]
      if (pt == 0 && it + 2 < n_my) {
        mbar_expect_tx(&sm.full_v[st], RB - 512); bulk_g2s(sm.rec_v[st], vrec + (size_t)(it + 2) * RB, RB - 512, &sm.full_v[st]);
      }
      if (pt == 0 && it + 3 < n_my) {
        mbar_expect_tx(&sm.full_va[it % 3], 512);
        bulk_g2s(sm.aux_v[it % 3], vrec + (size_t)(it + 3) * RB + (RB - 512), 512, &sm.full_va[it % 3]);
      }
    }
  } else if (warp >= 16) {
    // =============================== MMA issuer: one thread =========================================================
    if (warp == 16 && lane == 0) {
      auto issue_qk = [&](int c) {
        mbar_wait(&sm.kt_full[c & 1], (c >> 1) & 1);
        if (c > 0) mbar_wait(&sm.s_free, (c & 1) ^ 1);    // the softmax warps have read S of the previous chunk
        tc_fence_after();
#pragma unroll
        for (int term = 0; term < 2; ++term)
#pragma unroll
          for (int ks = 0; ks < DN_KT / 16; ++ks)
            umma_f16(tmem, umma_desc(smem_u32(term ? sm.qlo : sm.qhi) + ks * 256, 128, SBO_T),
                     umma_desc(smem_u32(sm.kt[c & 1]) + ks * 2 * DN_LBO, DN_LBO, DN_SBO_K), IDESC_S, (term | ks) != 0);
        if (c >= n_my) {                                  // raw chunk: + q'_hi x (second fp16 term of K, in the Vt buffer), N = 128
#pragma unroll
          for (int ks = 0; ks < DN_KT / 16; ++ks)
            umma_f16(tmem, umma_desc(smem_u32(sm.qhi) + ks * 256, 128, SBO_T),
                     umma_desc(smem_u32(sm.vt) + ks * 2 * DN_LBO, DN_LBO, DN_SBO_K), umma_idesc_f16(128, 128), 1u);
        }
        umma_commit(&sm.bar_s);
        umma_commit(&sm.k_free[c & 1]);
      };
      if (n_tot > 0) issue_qk(0);
      for (int it = 0; it < n_tot; ++it) {
        const uint32_t par = it & 1;
        const bool next_packed = it + 1 < n_my;           // a raw chunk's tiles exist only after this chunk's PV (see expand_k)
        if (next_packed) issue_qk(it + 1);                // runs while the softmax warps work on chunk it
        mbar_wait(&sm.vt_full, par);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          mbar_wait(&sm.p_full[h], par);
          tc_fence_after();
#pragma unroll
          for (int ks = 0; ks < DN_KPH / 16; ++ks) {      // 4 steps over the half's 64 tokens + 1 over the zero-point columns
            const uint32_t vcol = ks < 4 ? (uint32_t)(64 * h + 16 * ks) : 128u;
            umma_f16_ts(tmem + O_COL + 128 * h, tmem + P_COL + (DN_KPH / 2) * h + 8 * ks,
                        umma_desc(smem_u32(sm.vt) + (vcol >> 3) * DN_LBO, DN_LBO, DN_SBO_V), IDESC_O, (it | ks) != 0);
          }
          umma_commit(&sm.bar_o[h]);
        }
        if (!next_packed && it + 1 < n_tot) issue_qk(it + 1);
      }
    }
  } else {
    // =============================== softmax warps: thread = (query row = TMEM lane, token half) =====================
    setmaxnreg_inc<DENSE_REGS_SOFTMAX>();
    const int h = warp >> 2, r = (warp & 3) * 32 + lane;
    const uint32_t t_row = tmem + ((uint32_t)((warp & 3) * 32) << 16);
    const uint32_t t_o = t_row + O_COL + 128 * h;
    const uint32_t t_p = t_row + P_COL + (DN_KPH / 2) * h;
    // a warp whose 32 rows lie beyond the block's rows only keeps the barriers moving (its rows of P and O are never read)
    const bool live = rt * 128 + (warp & 3) * 32 < n_rows;
    const int i_tok = (rt * 128 + r) / g;                // query token of this row (causal mask of the block's own tokens)
    for (int it = 0; it < n_tot; ++it) {
      const int st = it % 3;
      const uint32_t par = it & 1;
      mbar_wait(&sm.bar_s, par);
      if (!live) {
        mbar_arrive_warp(&sm.s_free, lane);
        if (it > 0) mbar_wait(&sm.bar_o[h], par ^ 1);
        mbar_arrive_warp(&sm.p_full[h], lane);
        continue;
      }
      mbar_wait(&sm.aux_full[st], (it / 3) & 1);         // the producers' aux writes of this chunk are visible
      tc_fence_after();
      float2 v[32];                                      // logits of the half's 64 tokens, as token pairs
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
          for (int j = 0; j < 16; j += 2) v[(c0 + j) >> 1] = make_float2(__uint_as_float(u[j]), __uint_as_float(u[j + 1]));
        }
      }
      tc_fence_before();
      mbar_arrive_warp(&sm.s_free, lane);                         // S is in registers: the next QK^T may overwrite it
      const float2* as2 = &sm.aux_s2[st][32 * h];
      const float2* azm = &sm.aux_zm[st][32 * h];
      const float2 ec = sm.e_chunk[st];
      const float2 beta2 = make_float2(beta, beta), e2 = make_float2(ec.x, ec.x);
      float mxa[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
      {
        // aux in batches of 8 pairs, the next batch requested before this one is used
        const float4* as4 = reinterpret_cast<const float4*>(as2);
        float4 cur[4], nxt[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) cur[i] = as4[i];
#pragma unroll
        for (int bq = 0; bq < 4; ++bq) {
          if (bq < 3) {
#pragma unroll
            for (int i = 0; i < 4; ++i) nxt[i] = as4[4 * (bq + 1) + i];
          }
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int k = 8 * bq + 2 * i;
            v[k] = __ffma2_rn(make_float2(cur[i].x, cur[i].y), __fadd2_rn(v[k], beta2), e2);   // log2-domain logit of p~ = p 2^E
            v[k + 1] = __ffma2_rn(make_float2(cur[i].z, cur[i].w), __fadd2_rn(v[k + 1], beta2), e2);
            mxa[i] = fmaxf(mxa[i], fmaxf(fmaxf(v[k].x, v[k].y), fmaxf(v[k + 1].x, v[k + 1].y)));
          }
#pragma unroll
          for (int i = 0; i < 4; ++i) cur[i] = nxt[i];
        }
      }
      float mx = fmaxf(fmaxf(mxa[0], mxa[1]), fmaxf(mxa[2], mxa[3]));
      const int2 mk = sm.mask[st];
      if (mk.x < 128 || mk.y != DN_NO_MASK) {            // raw chunk (CTA-uniform): masked columns leave the softmax
        const int n_vis = min(mk.x, mk.y == DN_NO_MASK ? 128 : mk.y + i_tok + 1) - 64 * h;   // visible: columns 64 h + [0, n_vis)
        mx = -INFINITY;
#pragma unroll
        for (int k = 0; k < 32; ++k) {
          if (2 * k >= n_vis) v[k].x = -INFINITY;
          if (2 * k + 1 >= n_vis) v[k].y = -INFINITY;
          mx = fmaxf(mx, fmaxf(v[k].x, v[k].y));
        }
      }
      // (a row that has seen nothing yet keeps m_ref = -inf: every p~ is 2^(-inf - 0) = 0 and nothing is rescaled)
      const float m_cand = fmaxf(m_ref, mx - P_OFF);
      const float m_new = m_cand == -INFINITY ? 0.f : m_cand;
      const float f_old = ex2_approx(m_ref - m_new);     // 0 for the first chunk (m_ref = -inf)
      if (it > 0) {
        mbar_wait(&sm.bar_o[h], par ^ 1);                // PV of the previous chunk is complete: p~ of it may be overwritten, O is consistent
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
      m_ref = m_cand;
      const float2 nm2 = make_float2(-m_new, -m_new);
      float2 l2 = make_float2(0.f, 0.f), z2 = make_float2(0.f, 0.f);
#pragma unroll
      for (int c0 = 0; c0 < 32; c0 += 16) {              // 16 token pairs = 16 columns of the row's p~ in tensor memory
        uint32_t o[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) {
          const float2 d = __fadd2_rn(v[c0 + k], nm2);
          const __half2 ph = __floats2half2_rn(ex2_approx(d.x), ex2_approx(d.y));
          const float2 pf = __half22float2(ph);                 // the rounded values: numerator and denominator agree
          l2 = __fadd2_rn(l2, pf);
          z2 = __ffma2_rn(pf, azm[c0 + k], z2);
          o[k] = *reinterpret_cast<const uint32_t*>(&ph);
        }
        tmem_st16(t_p + c0, o);
      }
      const float lsum = (l2.x + l2.y) * ec.y, zsum = z2.x + z2.y;   // l in units of p = p~ 2^-E
      l_run = fmaf(l_run, f_old, lsum);
      {
        const __half zh = __float2half_rn(zsum), zl = __float2half_rn(zsum - __half2float(zh));
        const __half2 zz = __halves2half2(zh, zl);                                         // K columns 64, 65; 66..79: zero
        const uint32_t o8[8] = {*reinterpret_cast<const uint32_t*>(&zz), 0u, 0u, 0u, 0u, 0u, 0u, 0u};
        tmem_st8(t_p + 32, o8);
      }
      asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
      tc_fence_before();
      mbar_arrive_warp(&sm.p_full[h], lane);
    }
    // ---- epilogue (softmax warps): the two token halves of a row are LSE-merged here (m = max, weights 2^(m_h - m)),
    //      O rows -> shared memory (the q tiles are dead: every QK^T has completed), inverse Hadamard; then either the
    //      normalised result (one CTA per row tile: splits == 1) or the partial {m, l, o[128]} of set `split` -----------
    float* stage = reinterpret_cast<float*>(sm.qhi);     // [128][128] fp32 = qhi + qlo
    float2* ml = sm.ml();                                // [0, 256): {m, l} of (half, row); [256, 384): merged
    ml[128 * h + r] = make_float2(m_ref, l_run);
    if (n_tot > 0) {
      mbar_wait(&sm.bar_o[h], (n_tot - 1) & 1);
      tc_fence_after();
    }
    softmax_sync();
    const float2 a0 = ml[r], a1 = ml[128 + r];
    const float m_row = fmaxf(a0.x, a1.x);
    const float w0 = a0.x == -INFINITY ? 0.f : ex2_approx(a0.x - m_row), w1 = a1.x == -INFINITY ? 0.f : ex2_approx(a1.x - m_row);
    const float w_me = h ? w1 : w0;
    if (h == 0) {
      ml[256 + r] = make_float2(m_row, fmaf(w0, a0.y, w1 * a1.y));
#pragma unroll 1
      for (int c0 = 0; c0 < 128; c0 += 16) {
        uint32_t u[16];
        if (n_tot > 0) tmem_ld16(t_o + c0, u);
#pragma unroll
        for (int j = 0; j < 16; j += 4) {
          float4 o4 = make_float4(0.f, 0.f, 0.f, 0.f);
          if (w_me > 0.f) o4 = make_float4(w_me * __uint_as_float(u[j]), w_me * __uint_as_float(u[j + 1]),
                                           w_me * __uint_as_float(u[j + 2]), w_me * __uint_as_float(u[j + 3]));
          *reinterpret_cast<float4*>(&stage[r * 128 + ((c0 + j) ^ ((r & 7) << 2))]) = o4;
        }
      }
    }
    softmax_sync();
    if (h == 1 && n_tot > 0) {                           // (warp-uniform: tcgen05.ld is a warp-wide instruction)
#pragma unroll 1
      for (int c0 = 0; c0 < 128; c0 += 16) {
        uint32_t u[16];
        tmem_ld16(t_o + c0, u);
        if (w_me > 0.f) {
#pragma unroll
          for (int j = 0; j < 16; j += 4) {
            float4* sp = reinterpret_cast<float4*>(&stage[r * 128 + ((c0 + j) ^ ((r & 7) << 2))]);
            float4 o4 = *sp;
            o4.x = fmaf(w_me, __uint_as_float(u[j]), o4.x); o4.y = fmaf(w_me, __uint_as_float(u[j + 1]), o4.y);
            o4.z = fmaf(w_me, __uint_as_float(u[j + 2]), o4.z); o4.w = fmaf(w_me, __uint_as_float(u[j + 3]), o4.w);
            *sp = o4;
          }
        }
      }
    }
    tc_fence_before();
    softmax_sync();
    const bool direct = A.splits == 1;
    for (int rr = warp; rr < 128; rr += 8) {
      const int R = rt * 128 + rr;
      if (R >= n_rows) break;
      const int i = R / g, hq = R - i * g;
      const size_t row = ((size_t)b * A.n_q + i) * A.Hq + hkv * g + hq;
      const float4 s4 = *reinterpret_cast<const float4*>(&stage[rr * 128 + ((4 * lane) ^ ((rr & 7) << 2))]);
      float v[4] = {s4.x, s4.y, s4.z, s4.w};
      if (A.rotate_v) {
        fwht128_lane4(v, lane);
#pragma unroll
        for (int j = 0; j < 4; ++j) v[j] *= 0.08838834764831845f;
      }
      const float2 mlr = ml[256 + rr];
      if (direct) {
        const float inv = mlr.y > 0.f ? 1.f / mlr.y : 0.f;     // an empty cache and an empty block: zeros
        if (A.out_dtype == KVARN_F32) {
          *reinterpret_cast<float4*>(reinterpret_cast<float*>(A.out) + row * D + 4 * lane) = make_float4(v[0] * inv, v[1] * inv, v[2] * inv, v[3] * inv);
        } else {
          const __nv_bfloat162 o01 = __floats2bfloat162_rn(v[0] * inv, v[1] * inv), o23 = __floats2bfloat162_rn(v[2] * inv, v[3] * inv);
          *reinterpret_cast<uint2*>(reinterpret_cast<__nv_bfloat16*>(A.out) + row * D + 4 * lane) =
              make_uint2(*reinterpret_cast<const uint32_t*>(&o01), *reinterpret_cast<const uint32_t*>(&o23));
        }
      } else {
        float* prow = A.parts + ((size_t)split * ((size_t)A.B * A.n_q * A.Hq) + row) * PART_STRIDE;
        *reinterpret_cast<float4*>(prow + 4 + 4 * lane) = make_float4(v[0], v[1], v[2], v[3]);
        if (lane == 0) *reinterpret_cast<float4*>(prow) = make_float4(mlr.x, mlr.y, 0.f, 0.f);
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(TMEM_COLS));
}

}  // namespace kvarn

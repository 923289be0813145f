// kvarn_decode_attention for sm_100a: split-K over 128-token chunks; every warp stages whole records with its own
// TMA bulk copies into its own shared-memory slots; the two g x 128 x 128 contractions of every chunk run on the
// tensor cores as integer MMAs straight on the packed codes; split partials merge through distributed shared
// memory inside a thread-block cluster.  SURVEY 8(a) rows D1-D7; DESIGN.md "Decode kernel".
//
//   D1  q' = (q H / sqrt(128)) * sm_scale * log2(e)                    (online Q transform)
//   D2  record (codes + aux) -> shared memory, cp.async.bulk + mbarrier
//   D3  qt[h,c] = q'[h,c] s1[c];  beta[h] = sum_c qt[h,c] z[c]
//       logit[h,t] = s2[t] (sum_c qt[h,c] code[t,c] + beta[h])          (Eq. 1)
//   D4  online softmax in the log2 domain
//   D5  pt[h,t] = p[h,t] s1v[t];  a[h,c] = sum_t pt[h,t] (codeV[t,c] + zv[t]);  acc[h,c] += s2v[c] a[h,c]
//   D6  residual window: raw tokens in the un-rotated space
//   D7  split partials: reduce-scatter by head through DSMEM inside the cluster (and through
//       the workspace when several clusters share a sequence), inverse Hadamard, normalise.
//
// How the contractions reach the tensor cores without a dequantised tile
// ---------------------------------------------------------------------
// A operand = the codes themselves (u8): a thread expands the packed words of its
// MMA rows (K tile: tokens, V tile: channels) with ONE LOP3 per four codes,
//     reg(kappa) = W & (MASK0 << BITS*j(kappa)),
// i.e. a code stays where it is inside its byte and carries the factor 2^(BITS*j),
// the same for every code of k-step kappa.  The B operand compensates: the
// fixed-point value of qt (or pt) at that K position is multiplied by
// CLSMAX / 2^(BITS*j) before it is split into radix-256 digits (s8 digits for qt,
// u8 digits for pt).  Each digit plane is one B column, so the MMA yields, per
// token, the exact int32 sums  D[t][(h, i)] = sum_k A[t,k] * digit_i(X[h,k])  and
//     sum_c Q[h,c] code[t,c] = (sum_i 256^i D[t][(h,i)]) / CLSMAX   exactly.
// The only rounding is the fixed-point conversion of qt (relative to max_c |qt[h,c]|) and of
// pt (relative to the chunk's largest pt); beta and the zero-point term of V use the same
// values, so no cancellation error appears between the code term and the zero-point term.
// The two-plane ("aligned") form of the operands is described at decode_kernel_w.
//
// Why warp-level mma.sync (IMMA m16n8k32) and not tcgen05: the contraction is tiny
// (N = digits x g heads <= 32 columns) and the kernel is bound by instruction issue, not by
// tensor throughput; tcgen05 would also tie a 128-row accumulator to all four warps of a CTA
// (a warp reads only its own 32 TMEM lanes), i.e. bring back the CTA barriers per chunk that
// the warp-private pipelines remove.  The round-1 tcgen05 variant of this kernel is measured
// in DESIGN.md 6.2 (history); the dense multi-token kernel is where tcgen05 belongs.
#pragma once

#include <type_traits>

#include "kvarn_common.cuh"

namespace kvarn {

constexpr int WS_STRIDE = 260;  // floats per partial: m, l, pad, pad, acc_rot[128], acc_res[128]
constexpr int PART_STRIDE = 132;  // floats per exported partial (kvarn_decode_attention_partial): m, l, pad, pad, o[128]

struct DecodeArgs {
  const uint8_t* k_records;
  const uint8_t* v_records;
  const void* k_resid;
  const void* v_resid;
  const void* k_sink;   // [B][Hkv][n_sink][128] raw sink tokens, or null
  const void* v_sink;
  int n_sink;
  const int32_t* seq_lens;
  int32_t* ticket;  // [B*Hkv], zero between calls (self-resetting)
  const void* q;
  void* out;
  float* ws;
  int B, Hkv, Hq, g, max_chunks, splits;
  int cluster;    // CTAs per thread-block cluster along the split axis (1..16): merged through DSMEM
  int nclus;      // clusters per (sequence, KV head); splits = cluster * nclus; nclus > 1 -> workspace merge
  float q_scale;  // sm_scale * log2(e)
  int rotate_k, rotate_v, out_dtype;
  // multi-token read path (kvarn_block_attention, Fig. 4): n_q query tokens per sequence, q / out
  // [B][n_q][Hq][128]; blockIdx.z picks `tpc` of them, whose tpc * g (token, head) pairs are the MMA
  // columns of the CTA.  k_blk / v_blk [B][Hkv][n_q][128]: the block's own raw tokens, attended
  // causally (query i sees block tokens 0..i).  Plain decode: n_q = tpc = 1, k_blk = null.
  int n_q, tpc;
  const void* k_blk;
  const void* v_blk;
  // context-parallel building block: 1 = write the un-normalised partial {m, l, o[128]} of every (b, q head) to
  // `out` ([B][Hq][PART_STRIDE] fp32) instead of the normalised output; merged across ranks by merge_partials_kernel
  int partial;
  // 4, 16, 64: the plane shifts of the aligned A fragments as MULTIPLIERS from the constant bank -- an integer
  // multiply issues on the fma pipe, and only an operand ptxas cannot see through keeps it from becoming a shift
  // on the alu pipe (the busiest unit of the 2-bit kernel)
  uint32_t shl_mul[3];
  // 1: leave the packed chunks to another kernel (block_dense_kernel) and run the raw windows only
  int skip_chunks;
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

// thread-block cluster: rank, peer shared-memory addresses (DSMEM), barrier
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t mapa_shared(uint32_t saddr, uint32_t cta_rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(cta_rank));
  return r;
}
__device__ __forceinline__ void st_cluster_f32(uint32_t addr, float v) {
  asm volatile("st.shared::cluster.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

// D (s32, 16x8) += A (u8 or s8, 16x32, row) * B (s8 or u8, 32x8, col)
template <bool B_SIGNED, bool A_SIGNED = false>
__device__ __forceinline__ void imma_16832(int32_t (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  if (A_SIGNED)   // (only with signed B: the centred-code form of the QK^T contraction)
    asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.s8.s8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+r"(d[0]), "+r"(d[1]), "+r"(d[2]), "+r"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
  else if (B_SIGNED)
    asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.u8.s8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+r"(d[0]), "+r"(d[1]), "+r"(d[2]), "+r"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
  else
    asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.u8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+r"(d[0]), "+r"(d[1]), "+r"(d[2]), "+r"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel) {
  uint32_t r;
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(sel));
  return r;
}
// 4x4 byte transpose: y[d] = (byte d of x[0], x[1], x[2], x[3])
__device__ __forceinline__ void transpose4x4(const uint32_t (&x)[4], uint32_t (&y)[4]) {
  const uint32_t t0 = prmt(x[0], x[1], 0x5140), t1 = prmt(x[2], x[3], 0x5140);
  const uint32_t t2 = prmt(x[0], x[1], 0x7362), t3 = prmt(x[2], x[3], 0x7362);
  y[0] = prmt(t0, t1, 0x5410); y[1] = prmt(t0, t1, 0x7632);
  y[2] = prmt(t2, t3, 0x5410); y[3] = prmt(t2, t3, 0x7632);
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
// red_index<NV>(lane) -- every index is held by 32/NV lanes.  (Residual window.)
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

// single-instruction MUFU forms (no denormal / range fix-up code around them)
__device__ __forceinline__ float ex2_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rcp_approx(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float lg2_approx(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

constexpr float MAGIC_F = 12582912.0f;       // 1.5 * 2^23: (x + MAGIC) rounds x to an integer (RNE) for |x| <= 2^22
constexpr int MAGIC_I = 0x4B400000;
constexpr float Q_FIX = 4194300.0f;          // 2^22: fixed-point scale of qt relative to max_c |qt[h,c]|
constexpr float P_FIX = 4194304.0f;          // 2^22: fixed-point scale of pt = p s1v <= 1

// 16-byte slot of fragment lane lane' inside a [nu][hk] block of a B operand: bit 2 is flipped by
// (bit 3 of lane') ^ hk, which spreads the builders' 32-bit stores over twice as many banks and keeps
// the fragment loads (one LDS.128 per lane) conflict-free
__device__ __forceinline__ int b_slot(int lane_p, int hk) { return lane_p ^ ((((lane_p >> 3) ^ hk) & 1) << 2); }

// Packed words of the four MMA rows (mtile mt; rho = 0, 1) this thread feeds: W[rho][word]
template <int BITS>
__device__ __forceinline__ void load_row_words(const uint8_t* codes, int warp, int lane, int mt, uint32_t (&W)[2][BITS == 2 ? 2 : 4]) {
  if constexpr (BITS == 2) {
    const uint4 v = *reinterpret_cast<const uint4*>(codes + warp * 1024 + mt * 512 + lane * 16);
    W[0][0] = v.x; W[0][1] = v.y; W[1][0] = v.z; W[1][1] = v.w;
  } else {
#pragma unroll
    for (int rho = 0; rho < 2; ++rho) {
      const uint4 v = *reinterpret_cast<const uint4*>(codes + warp * 2048 + mt * 1024 + rho * 512 + lane * 16);
      W[rho][0] = v.x; W[rho][1] = v.y; W[rho][2] = v.z; W[rho][3] = v.w;
    }
  }
}
// A fragment of k-step kappa: one LOP3 per register
template <int BITS>
__device__ __forceinline__ void a_frag(const uint32_t (&W)[2][BITS == 2 ? 2 : 4], int kappa, uint32_t (&a)[4]) {
  constexpr uint32_t MASK0 = BITS == 2 ? 0x03030303u : 0x0F0F0F0Fu;
  const int j = BITS == 2 ? kappa : (kappa & 1);
  const int w0 = BITS == 2 ? 0 : 2 * (kappa >> 1);
  const uint32_t m = MASK0 << (BITS * j);
  a[0] = W[0][w0] & m; a[1] = W[1][w0] & m; a[2] = W[0][w0 + 1] & m; a[3] = W[1][w0 + 1] & m;
}

// radix-256 digits (d0 + 256 d1 + 65536 d2 + 2^24 d3) of the int32 sums -> float
__device__ __forceinline__ float undigit(int d0, int d1, int d2, int d3) {
  const int x01 = d1 * 256 + d0;
  const int x23 = d3 * 256 + d2;
  return fmaf(__int2float_rn(x23), 65536.f, __int2float_rn(x01));
}

// Columns of a CTA: j -> (query token tok0 + (j >> lg), head j mod 2^lg); plain decode: tok0 = 0, ncols = g, lg = 31
// (column = head, any g).  Evaluated once before and once after the main loop -- the volatile read of %ctaid.z
// keeps the two evaluations apart, so that none of this lives in registers through the loop (at g = 8 the loop is
// register-bound: carrying these values cost 6 % more loop instructions).
// Which (sequence, KV head, split) this CTA serves and the regions of its sequence (sink | body | residual);
// like col_map, evaluated before and after the main loop from volatile reads so nothing is carried through it.
struct Where { int bh, b, hkv, split, n_sink_tok, n_chunks, resid; };
// AGAIN = false: the plain form (blockIdx, an ordinary load: the compiler keeps these in uniform registers);
// AGAIN = true: volatile reads, a second evaluation the compiler cannot merge with the first.
template <bool AGAIN>
__device__ __forceinline__ Where where_am_i(const DecodeArgs& A) {
  unsigned x = blockIdx.x, y = blockIdx.y;
  if constexpr (AGAIN) {
    asm volatile("mov.u32 %0, %%ctaid.x;" : "=r"(x));
    asm volatile("mov.u32 %0, %%ctaid.y;" : "=r"(y));
  }
  Where w;
  w.bh = (int)x; w.b = w.bh / A.Hkv; w.hkv = w.bh - w.b * A.Hkv; w.split = (int)y;
  int len;
  if constexpr (AGAIN) asm volatile("ld.global.cg.s32 %0, [%1];" : "=r"(len) : "l"(A.seq_lens + w.b));
  else len = A.seq_lens[w.b];
  w.n_sink_tok = min(len, A.n_sink);
  const int body = len - w.n_sink_tok;
  w.n_chunks = min(body >> 7, A.max_chunks);
  w.resid = body & 127;
  return w;
}

struct ColMap { int lg, tok0, ncols, n_q, blk_cnt; };
template <bool AGAIN>
__device__ __forceinline__ ColMap col_map(const DecodeArgs& A) {
  unsigned z = blockIdx.z;
  if constexpr (AGAIN) asm volatile("mov.u32 %0, %%ctaid.z;" : "=r"(z));
  ColMap c;
  c.lg = A.tpc == 1 ? 31 : __ffs(A.g) - 1;
  c.n_q = A.n_q;
  c.tok0 = (int)z * A.tpc;
  c.ncols = min(A.tpc, c.n_q - c.tok0) * A.g;
  c.blk_cnt = A.k_blk != nullptr ? min(c.n_q, c.tok0 + A.tpc) : 0;   // block tokens visible to some column of this CTA
  return c;
}

// Slice `split` of a raw window of cnt tokens cut over n_splits CTAs (>= RAW_SLICE_MIN tokens per slice): first token, count.
constexpr int RAW_SLICE_MIN = 16;
__device__ __forceinline__ void raw_slice(int cnt, int split, int n_splits, int& t0, int& n) {
  t0 = 0; n = 0;
  if (cnt <= 0) return;                      // (no window: no integer division either)
  int per_w = (cnt + n_splits - 1) / n_splits;
  per_w = per_w < RAW_SLICE_MIN ? RAW_SLICE_MIN : per_w;
  t0 = split * per_w;
  n = min(max(cnt - t0, 0), per_w);
}
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
// the n rows (128 values each) at `base` towards L2: one 128-byte line per thread and step
template <typename InT>
__device__ __forceinline__ void prefetch_rows(const InT* base, int n, int tid) {
  const char* p = reinterpret_cast<const char*>(base);
  const int bytes = n * D * (int)sizeof(InT);
  for (int o = tid * 128; o < bytes; o += 128 * 128) prefetch_l2(p + o);
}

// ---- D6 + D7 of one CTA, shared by both main-loop variants: raw windows, merge of the split partials, finish.
// On entry thread tid = channel tid holds, per column h: m_run[h] (running maximum of the chunks, CTA-wide),
// l_tot[h] (l of the chunks, CTA-wide), l_part[h] (thread 0: l_tot, others 0) and acc[h] (its channel of the
// rotated accumulator).  `land` = the CTA's dead record ring (>= 16 x WS_STRIDE floats; the CTA has already done
// cluster_arrive()), `wsp` = >= GP x 64 floats of dead shared memory, `qraw` = [GP][128] q * q_scale (un-rotated; read by the raw windows,
// scratch afterwards).  SM needs qrot, hs, hz, wmax, wz, last_flag.
template <int GP, typename InT, class SM>
__device__ __forceinline__ void decode_finish(const DecodeArgs& A, SM& sm, float* land, float* wsp, float* qraw, const Where& w1,
                                              const ColMap& cm, const bool do_resid, const bool do_sink,
                                              float (&m_run)[GP], float (&l_part)[GP], float (&l_tot)[GP], float (&acc)[GP]) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = A.g;
  const int bh = w1.bh, b = w1.b, hkv = w1.hkv, split = w1.split, n_sink_tok = w1.n_sink_tok, resid = w1.resid;
  const int lg = cm.lg, tok0 = cm.tok0, ncols = cm.ncols, n_q = cm.n_q, blk_cnt = cm.blk_cnt;
  const bool has_blk = A.k_blk != nullptr;
  // Every raw window (sink, residual, the block's own tokens) is cut into A.splits slices of >= RAW_SLICE_MIN tokens, one
  // per CTA of the (sequence, KV head): a window's cost is the latency of its dependent global loads (thread = token, few
  // warps), so slices run side by side instead of one CTA walking 128 tokens; the partials merge like the chunks'.
  int sink_t0, sink_n, res_t0, res_n, blk_t0, blk_n;
  raw_slice(n_sink_tok, split, A.splits, sink_t0, sink_n);
  raw_slice(resid, split, A.splits, res_t0, res_n);
  raw_slice(has_blk ? blk_cnt : 0, split, A.splits, blk_t0, blk_n);
  const bool ran_raw = (sink_n | res_n | blk_n) > 0;                 // CTA-uniform
  const bool any_raw = n_sink_tok > 0 || resid > 0 || has_blk;       // uniform over the CTAs of this (sequence, KV head)
  (void)do_resid; (void)do_sink;
  auto qrow = [&](int j) -> size_t { return ((size_t)b * n_q + tok0 + (j >> lg)) * A.Hq + hkv * g + (j - ((j >> lg) << lg)); };
  // ---- D6: raw windows (sink tokens of split 0, residual window of the last split; un-rotated space) ----
  float acc_res[GP];
#pragma unroll
  for (int h = 0; h < GP; ++h) acc_res[h] = 0.f;
  float* psm = &sm.qrot[0][0];   // [GP][128] probabilities of the window (q' and the staged acc are dead by now)
  // vis0: token tid is visible to column h iff tid <= vis0 + (h >> lg) (causal block); NO_MASK for sink / residual
  constexpr int NO_MASK = 1 << 20;
  auto raw_window = [&](const InT* kraw, const InT* vraw, const int cnt, const int vis0) {   // cnt <= 128 tokens, thread = token
    float logit[GP];
#pragma unroll
    for (int h = 0; h < GP; ++h) logit[h] = 0.f;
    if (tid < cnt) {
      const InT* row = kraw + (size_t)tid * D;
      constexpr int CB = 64;   // channels per batch: all loads of a batch are in flight together
#pragma unroll 1
      for (int c0 = 0; c0 < D; c0 += CB) {
        float kv[CB / 8][8];
#pragma unroll
        for (int j = 0; j < CB / 8; ++j) ld_in8(row + c0 + 8 * j, kv[j]);
#pragma unroll
        for (int j = 0; j < CB / 8; ++j) {
          const int c = c0 + 8 * j;
#pragma unroll
          for (int h = 0; h < GP; ++h) {
            const float4 q0 = *reinterpret_cast<const float4*>(&qraw[h * 128 + c]);
            const float4 q1 = *reinterpret_cast<const float4*>(&qraw[h * 128 + c + 4]);
            float s = logit[h];
            s = fmaf(kv[j][0], q0.x, s); s = fmaf(kv[j][1], q0.y, s); s = fmaf(kv[j][2], q0.z, s); s = fmaf(kv[j][3], q0.w, s);
            s = fmaf(kv[j][4], q1.x, s); s = fmaf(kv[j][5], q1.y, s); s = fmaf(kv[j][6], q1.z, s); s = fmaf(kv[j][7], q1.w, s);
            logit[h] = s;
          }
        }
      }
    } else {
#pragma unroll
      for (int h = 0; h < GP; ++h) logit[h] = -INFINITY;
    }
    if (vis0 != NO_MASK) {
#pragma unroll
      for (int h = 0; h < GP; ++h) if (tid > vis0 + (h >> lg)) logit[h] = -INFINITY;
    }
    {
      float v[GP];
#pragma unroll
      for (int h = 0; h < GP; ++h) v[h] = logit[h];
      const float r = warp_reduce_multi<GP>(v, lane, RMax());
      if ((lane & (32 / GP - 1)) == 0) sm.wmax[warp][red_index<GP>(lane)] = r;
    }
    __syncthreads();   // also: the previous window's probabilities have been consumed
    float p[GP];
#pragma unroll
    for (int h = 0; h < GP; ++h) {
      const float mc = fmaxf(fmaxf(sm.wmax[0][h], sm.wmax[1][h]), fmaxf(sm.wmax[2][h], sm.wmax[3][h]));
      const float m_new = fmaxf(m_run[h], mc);
      // (a column that has seen nothing yet and sees nothing of this slice either -- a causal slice beyond its query
      //  token in a CTA without chunks -- keeps m = -inf: no NaN from -inf - -inf)
      const float corr = m_new == -INFINITY ? 1.f : exp2f(m_run[h] - m_new);
      m_run[h] = m_new;
      p[h] = m_new == -INFINITY ? 0.f : exp2f(logit[h] - m_new);        // exp2(-inf) = 0 for masked tokens
      l_part[h] = fmaf(l_part[h], corr, p[h]);
      acc[h] *= corr;
      acc_res[h] *= corr;
      psm[h * 128 + tid] = p[h];
    }
    __syncthreads();
    constexpr int TB = 32;   // tokens per batch of the value pass (32 loads in flight per thread)
#pragma unroll 1
    for (int tb = 0; tb < cnt; tb += TB) {
      float vv[TB];
#pragma unroll
      for (int j = 0; j < TB; ++j) vv[j] = (tb + j < cnt) ? ld_in<InT>(vraw + (size_t)(tb + j) * D + tid) : 0.f;
#pragma unroll
      for (int j8 = 0; j8 < TB; j8 += 8) {
#pragma unroll
        for (int h = 0; h < GP; ++h) {
          const float4 p0 = *reinterpret_cast<const float4*>(&psm[h * 128 + tb + j8]);
          const float4 p1 = *reinterpret_cast<const float4*>(&psm[h * 128 + tb + j8 + 4]);
          float s = acc_res[h];
          s = fmaf(p0.x, vv[j8], s); s = fmaf(p0.y, vv[j8 + 1], s); s = fmaf(p0.z, vv[j8 + 2], s); s = fmaf(p0.w, vv[j8 + 3], s);
          s = fmaf(p1.x, vv[j8 + 4], s); s = fmaf(p1.y, vv[j8 + 5], s); s = fmaf(p1.z, vv[j8 + 6], s); s = fmaf(p1.w, vv[j8 + 7], s);
          acc_res[h] = s;
        }
      }
    }
    __syncthreads();   // psm and wmax are free again
  };
  if (sink_n > 0)
    raw_window(reinterpret_cast<const InT*>(A.k_sink) + ((size_t)bh * A.n_sink + sink_t0) * D,
               reinterpret_cast<const InT*>(A.v_sink) + ((size_t)bh * A.n_sink + sink_t0) * D, sink_n, NO_MASK);
  if (res_n > 0)
    raw_window(reinterpret_cast<const InT*>(A.k_resid) + ((size_t)bh * G + res_t0) * D,
               reinterpret_cast<const InT*>(A.v_resid) + ((size_t)bh * G + res_t0) * D, res_n, NO_MASK);
  if (blk_n > 0)       // causal: block token blk_t0 + tid is visible to query token i iff blk_t0 + tid <= i
    raw_window(reinterpret_cast<const InT*>(A.k_blk) + ((size_t)bh * n_q + blk_t0) * D,
               reinterpret_cast<const InT*>(A.v_blk) + ((size_t)bh * n_q + blk_t0) * D, blk_n, tok0 - blk_t0);

  // ---- l: reduce the per-thread partial sums (only a CTA that ran a raw window has any beyond the chunks') ----
  if (ran_raw) {   // CTA-uniform
    __syncthreads();
    {
      float v[GP];
#pragma unroll
      for (int h = 0; h < GP; ++h) v[h] = l_part[h];
      const float r = warp_reduce_multi<GP>(v, lane, RAdd());
      if ((lane & (32 / GP - 1)) == 0) sm.wz[warp][red_index<GP>(lane)] = r;
    }
    __syncthreads();
#pragma unroll
    for (int h = 0; h < GP; ++h) l_tot[h] = (sm.wz[0][h] + sm.wz[1][h]) + (sm.wz[2][h] + sm.wz[3][h]);
  }

  // ---- D7a: in-cluster merge of the split partials through distributed shared memory ----------
  // Reduce-scatter by head: head h is merged by the CTA of cluster rank h % CS, which receives the
  // partial of rank r in landing slot (h / CS) * CS + r.  The landing area is the record ring, dead
  // once every CTA of the cluster has left its main loop (first cluster barrier).  Afterwards this
  // CTA holds, in array slot j, the merged (m, l, acc, acc_res) of its owned head h = hbase + hstride j.
  const int CS = A.cluster, NC = A.nclus;
  int hbase = 0, hstride = 1;
  if (CS > 1) {
    const int crank = (int)cluster_ctarank();
        cluster_wait();
    const uint32_t land_addr = smem_u32(land);
#pragma unroll
    for (int h = 0; h < GP; ++h) {
      if (h < ncols) {
        const int j = h / CS, d = h - j * CS;
        const uint32_t dst = mapa_shared(land_addr + (uint32_t)(j * CS + crank) * (WS_STRIDE * 4), (uint32_t)d);
        if (tid == 0) { st_cluster_f32(dst, m_run[h]); st_cluster_f32(dst + 4, l_tot[h]); }
        st_cluster_f32(dst + 16 + 4 * tid, acc[h]);
        if (any_raw) st_cluster_f32(dst + 16 + 512 + 4 * tid, acc_res[h]);
      }
    }
    cluster_sync_all();
#pragma unroll
    for (int j = 0; j < GP; ++j) {
      const int h = crank + j * CS;
      float mj = -INFINITY, lj = 0.f, aj = 0.f, rj = 0.f;
      if (h < ncols) {
        const float* slot0 = land + j * CS * WS_STRIDE;
        for (int r = 0; r < CS; ++r) mj = fmaxf(mj, slot0[r * WS_STRIDE]);
        for (int r = 0; r < CS; ++r) {
          const float* sl = slot0 + r * WS_STRIDE;
          const float w = (sl[0] == -INFINITY) ? 0.f : ex2_approx(sl[0] - mj);
          lj = fmaf(w, sl[1], lj);
          aj = fmaf(w, sl[4 + tid], aj);
          if (any_raw) rj = fmaf(w, sl[132 + tid], rj);
        }
      }
      m_run[j] = mj; l_tot[j] = lj; acc[j] = aj; acc_res[j] = rj;
    }
    hbase = crank; hstride = CS;
    if (hbase >= ncols) return;   // this rank owns no column
  }

  // ---- D7b: several clusters per (sequence, KV head): partials -> workspace, last arriver merges ----
  if (NC > 1) {
    const int cidx = split / CS;
#pragma unroll
    for (int j = 0; j < GP; ++j) {
      const int h = hbase + hstride * j;
      if (h < ncols) {
        float* o = A.ws + (qrow(h) * NC + cidx) * WS_STRIDE;
        if (tid == 0) { o[0] = m_run[j]; o[1] = l_tot[j]; }
        o[4 + tid] = acc[j];
        o[132 + tid] = acc_res[j];
      }
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) {
      const int n_writers = NC * min(CS, ncols);   // CTAs that own at least one column
      int* tk = &A.ticket[(size_t)blockIdx.z * gridDim.x + bh];
      const int old = atomicAdd(tk, 1);
      const int last = (old == n_writers - 1);
      if (last) *tk = 0;
      sm.last_flag = last;
    }
    __syncthreads();
    if (!sm.last_flag) return;
    __threadfence();
    // weights of the partials: warp w handles heads w, w+4; lane s handles partials s, s+32
        for (int h = warp; h < ncols; h += 4) {
      const float* base = A.ws + qrow(h) * NC * WS_STRIDE;
      const float m0 = lane < NC ? __ldcg(base + (size_t)lane * WS_STRIDE) : -INFINITY;
      const float m1 = lane + 32 < NC ? __ldcg(base + (size_t)(lane + 32) * WS_STRIDE) : -INFINITY;
      const float l0 = lane < NC ? __ldcg(base + (size_t)lane * WS_STRIDE + 1) : 0.f;
      const float l1 = lane + 32 < NC ? __ldcg(base + (size_t)(lane + 32) * WS_STRIDE + 1) : 0.f;
      const float mstar = warp_max(fmaxf(m0, m1));
      const float w0 = (m0 == -INFINITY) ? 0.f : exp2f(m0 - mstar);
      const float w1 = (m1 == -INFINITY) ? 0.f : exp2f(m1 - mstar);
      wsp[h * 64 + lane] = w0;
      wsp[h * 64 + lane + 32] = w1;
      const float L = warp_sum(fmaf(w0, l0, w1 * l1));
      if (lane == 0) { sm.hs[0][h][1] = L; sm.hs[0][h][0] = mstar; }
    }
    __syncthreads();
#pragma unroll
    for (int h = 0; h < GP; ++h) {
      float rot = 0.f, res = 0.f, L = 0.f;
      if (h < ncols) {
        const float* base = A.ws + qrow(h) * NC * WS_STRIDE + 4 + tid;
        int s = 0;
        for (; s + 4 <= NC; s += 4) {
          float r[4], e[4];
#pragma unroll
          for (int j = 0; j < 4; ++j) { r[j] = __ldcg(base + (size_t)(s + j) * WS_STRIDE); e[j] = __ldcg(base + (size_t)(s + j) * WS_STRIDE + 128); }
#pragma unroll
          for (int j = 0; j < 4; ++j) { const float w = wsp[h * 64 + s + j]; rot = fmaf(w, r[j], rot); res = fmaf(w, e[j], res); }
        }
        for (; s < NC; ++s) {
          const float w = wsp[h * 64 + s];
          rot = fmaf(w, __ldcg(base + (size_t)s * WS_STRIDE), rot);
          res = fmaf(w, __ldcg(base + (size_t)s * WS_STRIDE + 128), res);
        }
        L = sm.hs[0][h][1];
        m_run[h] = sm.hs[0][h][0];
      }
      l_tot[h] = L; acc[h] = rot; acc_res[h] = res;
    }
    hbase = 0; hstride = 1;
  }

  // ---- D7c: inverse Hadamard, residual part, normalisation of the owned heads ---------------------
  float* merged_rot = &sm.qrot[0][0];   // [GP][128]
  __syncthreads();
#pragma unroll
  for (int j = 0; j < GP; ++j) {
    merged_rot[j * 128 + tid] = acc[j];
    qraw[j * 128 + tid] = (l_tot[j] > 0.f) ? acc_res[j] : 0.f;
    if (tid == 0) {
      sm.hs[0][j][0] = A.partial ? 1.f : ((l_tot[j] > 0.f) ? 1.f / l_tot[j] : 0.f);
      sm.hs[0][j][1] = (l_tot[j] > 0.f) ? m_run[j] : -INFINITY;
      sm.hz[0][j][0] = l_tot[j];
    }
  }
  __syncthreads();
  for (int jj = warp; jj < GP; jj += 4) {
    const int hh = hbase + hstride * jj;
    if (hh >= ncols) break;
    float4 r4 = *reinterpret_cast<const float4*>(&merged_rot[jj * 128 + 4 * lane]);
    float v[4] = {r4.x, r4.y, r4.z, r4.w};
    if (A.rotate_v) {
      fwht128_lane4(v, lane);
#pragma unroll
      for (int j = 0; j < 4; ++j) v[j] *= 0.08838834764831845f;
    }
    const float4 s4 = *reinterpret_cast<const float4*>(&qraw[jj * 128 + 4 * lane]);
    const float inv = sm.hs[0][jj][0];
    const float o0 = (v[0] + s4.x) * inv, o1 = (v[1] + s4.y) * inv, o2 = (v[2] + s4.z) * inv, o3 = (v[3] + s4.w) * inv;
    if (A.partial) {
      float* prow = reinterpret_cast<float*>(A.out) + qrow(hh) * PART_STRIDE;
      *reinterpret_cast<float4*>(prow + 4 + 4 * lane) = make_float4(o0, o1, o2, o3);
      if (lane == 0) *reinterpret_cast<float4*>(prow) = make_float4(sm.hs[0][jj][1], sm.hz[0][jj][0], 0.f, 0.f);
      continue;
    }
    const size_t off = qrow(hh) * D + 4 * lane;
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

// ======================================================================================================
// decode_kernel_w: the same D1-D7, with WARP-PRIVATE chunk pipelines.  Each of the CTA's 4 warps owns whole
// chunks (chunk c_begin + warp + 4 i): it stages the chunk's two records into its own shared-memory slots with
// its own TMA bulk copies / mbarriers, builds the B operands for all columns, contracts all 8 m-tiles and keeps
// a private online-softmax state (m, l, acc) -- no CTA barrier and no cross-warp exchange inside the loop, only
// __syncwarp.  The B fragments are loaded once per contraction and kept in registers, and the per-chunk
// reductions (maximum, zero-point sum) stay inside the warp.  K of the next chunk is requested as soon as the
// QK^T contraction has consumed the codes, V of the next chunk after the value contraction, so each slot is
// single-buffered (9.2 KB per warp at 2-bit).  After the loop the 4 private states are merged through the dead
// slots and the shared finish (decode_finish) runs as before.  Record layout and row-slot maps are unchanged:
// what was "warp" in slot s = 32 warp + 16 mtile + 8 rho + g is now the m-tile pair index mp of the owning warp.
//
// DQ / DP = radix-256 digit planes of the fixed-point q~ / p~.
//   4: the in-place A fragments of the CTA-cooperative variant (a code keeps its bit position 2j inside its byte,
//      the B operand carries 4^(3-j)): 22-bit values.
//   2: ALIGNED A fragments -- every plane is shifted to bits 7:6 of its byte ((W << 2 (3 - j)), an IMAD on the idle fma
//      pipe, then one LOP3), so all codes carry the same factor 64 and the B operand needs no compensation bits: two
//      digit planes hold 16 bits.  Half the columns: half the IMMAs, B-operand words, fragment loads and digit
//      recombinations.  For q~ (15 bits + sign, two balanced s8 digits) the A fragment is also CENTRED in the same
//      LOP3 (64 code - 96 as s8, i.e. code - 1.5) and beta = sum q~ (z + 1.5) takes the mean code in fp32, which removes
//      the mean part of the rounding error.  p~ with two u8 digits has 16 bits relative to the chunk's maximum.
// kvarn_params::decode_digits picks (DQ, DP): 0 (default) = (4, 2): 16-bit p~ costs < 1e-4 of the 2e-3 tolerance;
// 2 = (2, 2): fastest, q~ at 16 bits measured up to 1.2e-3 on short peaked contexts; 4 = (4, 4).
template <int BITS, int GP, int DQ, int DP>
struct WarpSm {
  static constexpr int RB = record_bytes(BITS);
  static constexpr int NTQ = GP * DQ / 8, NTP = GP * DP / 8;   // n-tiles (8 columns each): digit planes x GP columns
  static constexpr int NT = NTQ > NTP ? NTQ : NTP;
  alignas(128) uint8_t krec[RB];
  alignas(128) uint8_t vrec[RB];
  alignas(16) uint32_t bfr[NT][2][32][4];      // B fragments: first of q~ (QK^T), then -- reused -- of p~ (value contraction)
  alignas(16) float2 aux_a[128];               // per K row slot: {s2, log2 s1v}
  alignas(16) float2 aux_b[128];               //                 {1 / s1v, zv}
  alignas(8) __half aux_ch[4][8][4];           // per channel: s2v, [mp][fg][i] of channel slot 32 mp + 16 (i >> 1) + 8 (i & 1) + fg
  alignas(8) float2 hs[GP];                    // per column: {scale, beta}
  alignas(8) uint64_t fullk, fullv;
};
template <int BITS, int GP, int DQ, int DP>
struct DecSmemW {
  WarpSm<BITS, GP, DQ, DP> w[4];
  alignas(16) float qrot[GP][128];             // q' (rotated, scaled, in B-builder order); later p of a raw window / merged acc_rot
  alignas(16) float hs[1][GP][2];
  alignas(16) float hz[1][GP][4];
  alignas(16) float wmax[4][GP];
  alignas(16) float wz[4][GP];
  int last_flag;
};

// A fragment of k-step kappa, aligned form: the plane's codes moved to the top bits of their bytes, u8 value 64 code (16 code at 4-bit).
// CENTRED: s8 value 64 code - 96 = 64 (code - 1.5): bit 7 inverted, bit 6 kept, bit 5 set -- with M1 = bits {7, 5} and
// M2 = bits {6, 5} that is (M1 & ~M2 & ~x) | (~M1 & M2 & x) | (M1 & M2), one LOP3.
template <int BITS, bool CENTRED>
__device__ __forceinline__ void a_frag_aligned(const uint32_t (&W)[2][BITS == 2 ? 2 : 4], int kappa, uint32_t (&a)[4],
                                               const uint32_t (&shl_mul)[3]) {
  static_assert(BITS == 2 || !CENTRED, "centred A fragments: 2-bit records");
  constexpr int NCLS = 8 / BITS;
  constexpr uint32_t MASK = BITS == 2 ? 0xC0C0C0C0u : 0xF0F0F0F0u;
  const int j = BITS == 2 ? kappa : (kappa & 1);
  const int w0 = BITS == 2 ? 0 : 2 * (kappa >> 1);
  const int sh = BITS * (NCLS - 1 - j);      // compile-time per call site: 0, 2, 4 or 6
  auto f = [&](uint32_t w) -> uint32_t {
    const uint32_t x = sh == 0 ? w : w * shl_mul[sh / 2 - 1];
    if constexpr (!CENTRED) return x & MASK;
    constexpr uint32_t M1 = 0xA0A0A0A0u, M2 = 0x60606060u;
    return (M1 & ~M2 & ~x) | (~M1 & M2 & x) | (M1 & M2);
  };
  a[0] = f(W[0][w0]); a[1] = f(W[1][w0]); a[2] = f(W[0][w0 + 1]); a[3] = f(W[1][w0 + 1]);
}
template <int BITS, int NT, int NTB, bool B_SIGNED, bool ALIGNED, bool CENTRED = false>
__device__ __forceinline__ void contract_mp(const uint8_t* codes, const uint4 (&bf)[2][NTB], int mp, int lane, int32_t (&d)[2][NT][4],
                                            const uint32_t (&shl_mul)[3]) {
  uint32_t W[2][2][BITS == 2 ? 2 : 4];
  load_row_words<BITS>(codes, mp, lane, 0, W[0]);
  load_row_words<BITS>(codes, mp, lane, 1, W[1]);
#pragma unroll
  for (int mt = 0; mt < 2; ++mt)
#pragma unroll
    for (int nu = 0; nu < NT; ++nu)
#pragma unroll
      for (int c = 0; c < 4; ++c) d[mt][nu][c] = 0;
#pragma unroll
  for (int hk = 0; hk < 2; ++hk) {
#pragma unroll
    for (int k1 = 0; k1 < 2; ++k1) {
      const int kappa = 2 * hk + k1;
      uint32_t a[2][4];
      if constexpr (ALIGNED) { a_frag_aligned<BITS, CENTRED>(W[0], kappa, a[0], shl_mul); a_frag_aligned<BITS, CENTRED>(W[1], kappa, a[1], shl_mul); }
      else { a_frag<BITS>(W[0], kappa, a[0]); a_frag<BITS>(W[1], kappa, a[1]); }
#pragma unroll
      for (int nu = 0; nu < NT; ++nu)
#pragma unroll
        for (int mt = 0; mt < 2; ++mt) {
          if (k1) imma_16832<B_SIGNED, CENTRED>(d[mt][nu], a[mt], bf[hk][nu].z, bf[hk][nu].w);
          else imma_16832<B_SIGNED, CENTRED>(d[mt][nu], a[mt], bf[hk][nu].x, bf[hk][nu].y);
        }
    }
  }
}
// int32 digit sums of output (mt, i-th accumulator pair cc) of column u -> float
template <int DIG, int NT>
__device__ __forceinline__ float undigit_w(const int32_t (&dd)[2][NT][4], int mt, int u, int cc) {
  if constexpr (DIG == 4) return undigit(dd[mt][2 * u][cc], dd[mt][2 * u][cc + 1], dd[mt][2 * u + 1][cc], dd[mt][2 * u + 1][cc + 1]);
  else return __int2float_rn(dd[mt][u][cc + 1] * 256 + dd[mt][u][cc]);
}
constexpr float Q_FIX2 = 32639.0f;            // two planes: |Q| <= 2^15 - 1 - 128 keeps the high balanced digit inside s8
constexpr float P_FIX2 = 65535.0f;            // two planes: 16-bit p~

template <int BITS, int GP, int DQ, int DP, typename InT>
#ifndef KVARN_DECW_OCC4
#define KVARN_DECW_OCC4 4
#endif
__global__ void __launch_bounds__(128, BITS == 2 ? (GP == 4 ? KVARN_DECW_OCC4 : 3) : 2) decode_kernel_w(const DecodeArgs A) {
  using SM = DecSmemW<BITS, GP, DQ, DP>;
  using WS = WarpSm<BITS, GP, DQ, DP>;
  constexpr int RB = WS::RB, NTQ = WS::NTQ, NTP = WS::NTP;
  constexpr int NCLS = 8 / BITS;
  static_assert((DQ == 2 || DQ == 4) && (DP == 2 || DP == 4) && (BITS == 2 || DQ == 4), "digit planes");
  constexpr float CLS_INV = BITS == 2 ? (1.f / 64.f) : (1.f / 16.f);  // 1 / CLSMAX (every form scales a code by CLSMAX)
  constexpr float QF = DQ == 4 ? Q_FIX : Q_FIX2, PF = DP == 4 ? P_FIX : P_FIX2;
  constexpr float ZC = DQ == 2 ? 0.5f * (float)((1 << BITS) - 1) : 0.f;   // centred K codes: the mean code moves into beta
  constexpr int HPW = GP / 4;   // columns per thread in the softmax (h = ft + 4u)

  extern __shared__ __align__(128) uint8_t smem_raw[];
  SM& sm = *reinterpret_cast<SM*>(smem_raw);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int fg = lane >> 2, ft = lane & 3;
  const int g = A.g;
  WS& ws = sm.w[warp];
  // Programmatic dependent launch (the launch carries cudaLaunchAttributeProgrammaticStreamSerialization): the next
  // kernel of the stream may be made resident as soon as every CTA of this grid has started, and this grid's CTAs may
  // have become resident while the previous kernel was still running -- nothing of global memory is touched before
  // the wait (seq_lens, records, q, out, workspace and ticket all belong to earlier kernels until then).  Both
  // instructions are no-ops in a launch without the attribute.
  asm volatile("griddepcontrol.launch_dependents;");
  asm volatile("griddepcontrol.wait;" ::: "memory");

  const Where w0 = where_am_i<false>(A);
  const ColMap cm0 = col_map<false>(A);
  const bool do_resid = (w0.split == A.splits - 1) && w0.resid > 0;
  const bool do_sink = (w0.split == 0) && w0.n_sink_tok > 0;
  // ---- chunk range of this split (the raw windows are sliced over all the CTAs of the unit: decode_finish) ----
  const int w_sink = 0, w_res = 0;
  const int nch = A.skip_chunks ? 0 : w0.n_chunks;
  const int per = (nch + w_sink + w_res + A.splits - 1) / A.splits;
  const int c_begin = min(max(w0.split * per - w_sink, 0), nch);
  const int c_end = min(max((w0.split + 1) * per - w_sink, 0), nch);
  const int n_mine = (c_end - c_begin - warp + 3) >> 2;            // chunks of this warp: c_begin + warp + 4 i
  const uint8_t* krec = A.k_records + ((size_t)w0.bh * A.max_chunks + c_begin + warp) * RB;
  const uint8_t* vrec = A.v_records + ((size_t)w0.bh * A.max_chunks + c_begin + warp) * RB;

  // this CTA's slices of the raw windows go towards L2 now: decode_finish reads them with dependent loads, long after
  {
    int t0, n;
    raw_slice(w0.n_sink_tok, w0.split, A.splits, t0, n);
    if (n > 0) {
      prefetch_rows(reinterpret_cast<const InT*>(A.k_sink) + ((size_t)w0.bh * A.n_sink + t0) * D, n, tid);
      prefetch_rows(reinterpret_cast<const InT*>(A.v_sink) + ((size_t)w0.bh * A.n_sink + t0) * D, n, tid);
    }
    raw_slice(w0.resid, w0.split, A.splits, t0, n);
    if (n > 0) {
      prefetch_rows(reinterpret_cast<const InT*>(A.k_resid) + ((size_t)w0.bh * G + t0) * D, n, tid);
      prefetch_rows(reinterpret_cast<const InT*>(A.v_resid) + ((size_t)w0.bh * G + t0) * D, n, tid);
    }
    raw_slice(A.k_blk != nullptr ? cm0.blk_cnt : 0, w0.split, A.splits, t0, n);
    if (n > 0) {
      prefetch_rows(reinterpret_cast<const InT*>(A.k_blk) + ((size_t)w0.bh * cm0.n_q + t0) * D, n, tid);
      prefetch_rows(reinterpret_cast<const InT*>(A.v_blk) + ((size_t)w0.bh * cm0.n_q + t0) * D, n, tid);
    }
  }
  // ---- setup: the warp's barriers and first loads; q ---------------------------------------------------
  if (lane == 0) {
    mbar_init(&ws.fullk, 1); mbar_init(&ws.fullv, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if (n_mine > 0) {
      mbar_expect_tx(&ws.fullk, RB); bulk_g2s(ws.krec, krec, RB, &ws.fullk);
      mbar_expect_tx(&ws.fullv, RB); bulk_g2s(ws.vrec, vrec, RB, &ws.fullv);
    }
  }
  // B-builder role of a lane: lane = 8 kappa + 4 half + t' owns the four K positions p = 16 half + 4 t' + b of
  // k-step kappa, i.e. one 32-bit word of a B fragment per digit plane
  const int bk = lane >> 3, bhalf = (lane >> 2) & 1, btp = lane & 3;
  // D1: q' = (q H / sqrt(128)) * q_scale, stored in builder order: qrot[h][4 lane + bb] = q'[h][channel(lane, bb)]
  for (int hh = warp; hh < GP; hh += 4) {
    float v[4] = {0.f, 0.f, 0.f, 0.f};
    if (hh < cm0.ncols) {
      const size_t row = ((size_t)w0.b * cm0.n_q + cm0.tok0 + (hh >> cm0.lg)) * A.Hq + w0.hkv * g + (hh - ((hh >> cm0.lg) << cm0.lg));
      const InT* qp = reinterpret_cast<const InT*>(A.q) + row * D + 4 * lane;
#pragma unroll
      for (int j = 0; j < 4; ++j) v[j] = ld_in<InT>(qp + j) * A.q_scale;
    }
    if (A.rotate_k) {
      fwht128_lane4(v, lane);
#pragma unroll
      for (int j = 0; j < 4; ++j) v[j] *= 0.08838834764831845f;
    }
    // element e = 4 lane + j of q' goes to builder position kaux_of_elem(e) (the order of K.s1 / K.z in the record)
#pragma unroll
    for (int j = 0; j < 4; ++j) sm.qrot[hh][kaux_of_elem(BITS, 4 * lane + j)] = v[j];
  }
  __syncthreads();

  // destination of the builder's digit words for column h: n-tile DH (h >> 2) + (d >> 1), column slot g' = 2 (h & 3) + (d & 1)
  // of the fragment block [nt][hk = bk >> 1][b_slot(4 g' + btp, hk)][2 (bk & 1) + bhalf]
  const int jq = BITS == 2 ? bk : (bk & 1);
  const uint32_t mul_q = 1u << (BITS * (NCLS - 1 - jq));
  const uint32_t add_q = 0x80808080u - ((uint32_t)MAGIC_I * mul_q);
  uint32_t* const bq_base = &ws.bfr[0][bk >> 1][0][2 * (bk & 1) + bhalf];
  // softmax role: thread (fg, ft) sees, per m-tile pair mp, tokens slot = 32 mp + 16 mt + 8 rho + fg of columns ft + 4u;
  // these four tokens are K positions b = 2 mt + rho of word (kappa = mp, half = fg >> 2, t' = fg & 3) of the value contraction
  float mr[HPW], lp[HPW], ac[4][HPW][4];
#pragma unroll
  for (int u = 0; u < HPW; ++u) {
    mr[u] = -INFINITY; lp[u] = 0.f;
#pragma unroll
    for (int mp = 0; mp < 4; ++mp)
#pragma unroll
      for (int i = 0; i < 4; ++i) ac[mp][u][i] = 0.f;
  }

#pragma unroll 1
  for (int it = 0; it < n_mine; ++it) {
    const uint32_t par = it & 1;
    const bool more = it + 1 < n_mine;
    mbar_wait(&ws.fullk, par);
    // ---- phase A: B_q (digit planes of the fixed-point q~) and beta for every column; s2 of the K rows -------
    {
      const uint8_t* kr = ws.krec;
      const uint32_t s1w = *reinterpret_cast<const uint32_t*>(kr + s1_off(BITS) + 4 * lane);
      const uint2 zw = *reinterpret_cast<const uint2*>(kr + z_off(BITS) + 8 * lane);
      const float2 s01 = e4m3x2_to_f32x2((uint16_t)(s1w & 0xffff)), s23 = e4m3x2_to_f32x2((uint16_t)(s1w >> 16));
      const float2 z01 = __half22float2(*reinterpret_cast<const __half2*>(&zw.x));
      const float2 z23 = __half22float2(*reinterpret_cast<const __half2*>(&zw.y));
      const float2 zc01 = make_float2(z01.x + ZC, z01.y + ZC), zc23 = make_float2(z23.x + ZC, z23.y + ZC);
      float bsum[GP];
#pragma unroll
      for (int h = 0; h < GP; ++h) {
        const float4 qv = *reinterpret_cast<const float4*>(&sm.qrot[h][4 * lane]);
        const float2 q01 = __fmul2_rn(make_float2(qv.x, qv.y), s01), q23 = __fmul2_rn(make_float2(qv.z, qv.w), s23);
        const float qt[4] = {q01.x, q01.y, q23.x, q23.y};
        float amax = fmaxf(fmaxf(fabsf(qt[0]), fabsf(qt[1])), fmaxf(fabsf(qt[2]), fabsf(qt[3])));
        // beta uses the unrounded qt (and, with centred codes, z + 1.5: the mean code stays in fp32)
        const float2 bz = __ffma2_rn(q01, zc01, __fmul2_rn(q23, zc23));
        bsum[h] = bz.x + bz.y;
        amax = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(amax)));   // non-negative floats order like their bits
        const float inv = amax > 1e-30f ? QF * rcp_approx(amax) : 0.f;
        if constexpr (DQ == 4) {
          uint32_t X[4], Y[4];
#pragma unroll
          for (int r = 0; r < 4; ++r) {
            const float f = fmaf(qt[r], inv, MAGIC_F);                  // integer Q in the low mantissa bits
            X[r] = (__float_as_uint(f) * mul_q + add_q) ^ 0x80808080u;   // balanced s8 digits of Q << shift
          }
          transpose4x4(X, Y);   // Y[d] = digit d of the four K positions = one B-fragment word of column (h, d)
#pragma unroll
          for (int d = 0; d < 4; ++d)
            bq_base[(2 * (h >> 2) + (d >> 1)) * 256 + b_slot(4 * (2 * (h & 3) + (d & 1)) + btp, bk >> 1) * 4] = Y[d];
        } else {
          // Q + 128 in the low 16 mantissa bits; bytes 0, 1 ^ 0x0080 = the balanced digits (d0, d1): Q = d0 + 256 d1
          const float2 i2 = make_float2(inv, inv), mg = make_float2(MAGIC_F + 128.f, MAGIC_F + 128.f);
          const float2 f01 = __ffma2_rn(q01, i2, mg), f23 = __ffma2_rn(q23, i2, mg);
          const uint32_t X0 = __float_as_uint(f01.x) ^ 0x80u, X1 = __float_as_uint(f01.y) ^ 0x80u;
          const uint32_t X2 = __float_as_uint(f23.x) ^ 0x80u, X3 = __float_as_uint(f23.y) ^ 0x80u;
          const uint32_t t0 = prmt(X0, X1, 0x5140), t1 = prmt(X2, X3, 0x5140);
#pragma unroll
          for (int d = 0; d < 2; ++d)
            bq_base[(h >> 2) * 256 + b_slot(4 * (2 * (h & 3) + d) + btp, bk >> 1) * 4] = prmt(t0, t1, d ? 0x7632 : 0x5410);
        }
        if (lane == h) ws.hs[h].x = amax * (1.f / QF) * CLS_INV;   // logit = s2 * (acc * scale + beta)
      }
      const float bs = warp_reduce_multi<GP>(bsum, lane, RAdd());
      if ((lane & (32 / GP - 1)) == 0) ws.hs[red_index<GP>(lane)].y = bs;
      // s2 of the K rows (stored in row-slot order): 4 slots per lane
      const uint32_t s2w = *reinterpret_cast<const uint32_t*>(kr + s2_off(BITS) + 4 * lane);
      const float2 a01 = e4m3x2_to_f32x2((uint16_t)(s2w & 0xffff)), a23 = e4m3x2_to_f32x2((uint16_t)(s2w >> 16));
      ws.aux_a[4 * lane + 0].x = a01.x; ws.aux_a[4 * lane + 1].x = a01.y;
      ws.aux_a[4 * lane + 2].x = a23.x; ws.aux_a[4 * lane + 3].x = a23.y;
    }
    // (the V record's aux conversions sit here, ahead of the QK^T contraction they do not depend on: independent work
    //  for the scheduler while the tensor-core chains run; the V record was requested a whole iteration ago)
    mbar_wait(&ws.fullv, par);
    {   // aux of the V record: per-token (row-slot order) s1v, zv; per-channel s2v
      const uint8_t* vr = ws.vrec;
      const uint32_t s1w = *reinterpret_cast<const uint32_t*>(vr + s1_off(BITS) + 4 * lane);
      const uint2 zw = *reinterpret_cast<const uint2*>(vr + z_off(BITS) + 8 * lane);
      const uint32_t s2w = *reinterpret_cast<const uint32_t*>(vr + s2_off(BITS) + 4 * lane);
      const float2 s01 = e4m3x2_to_f32x2((uint16_t)(s1w & 0xffff)), s23 = e4m3x2_to_f32x2((uint16_t)(s1w >> 16));
      const float2 z01 = __half22float2(*reinterpret_cast<const __half2*>(&zw.x));
      const float2 z23 = __half22float2(*reinterpret_cast<const __half2*>(&zw.y));
      const float s1v[4] = {s01.x, s01.y, s23.x, s23.y}, zv[4] = {z01.x, z01.y, z23.x, z23.y};
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const float s = fmaxf(s1v[j], 9.094947e-13f);   // 2^-40: a zero scale stays harmless
        // pt = p s1v = exp2(logit + log2 s1v - m): the maximum is taken over the shifted logits, so pt <= 1
        ws.aux_a[4 * lane + j].y = lg2_approx(s);
        ws.aux_b[4 * lane + j] = make_float2(rcp_approx(s), zv[j]);
      }
      {   // s2v of channels 4 lane + j (exact in fp16): channel slot c -> [c >> 5][c & 7][(c >> 3) & 3]
        uint32_t h2[2];
        asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h2[0]) : "h"((uint16_t)(s2w & 0xffff)));
        asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h2[1]) : "h"((uint16_t)(s2w >> 16)));
        const __half* hv = reinterpret_cast<const __half*>(h2);
#pragma unroll
        for (int j = 0; j < 4; ++j) ws.aux_ch[lane >> 3][4 * (lane & 1) + j][(lane >> 1) & 3] = hv[j];
      }
    }
    __syncwarp();
    // ---- D3: QK^T over the 8 m-tiles: raw integer sums -> float (the scales follow once V's aux is there) ----
    float sraw[4][HPW][4];
    {
      uint4 bf[2][NTQ];
#pragma unroll
      for (int hk = 0; hk < 2; ++hk)
#pragma unroll
        for (int nu = 0; nu < NTQ; ++nu) bf[hk][nu] = *reinterpret_cast<const uint4*>(&ws.bfr[nu][hk][b_slot(lane, hk)][0]);
#pragma unroll
      for (int mp = 0; mp < 4; ++mp) {
        int32_t dd[2][NTQ][4];
        contract_mp<BITS, NTQ, NTQ, true, DQ == 2, DQ == 2>(ws.krec, bf, mp, lane, dd, A.shl_mul);
#pragma unroll
        for (int u = 0; u < HPW; ++u)
#pragma unroll
          for (int i = 0; i < 4; ++i) sraw[mp][u][i] = undigit_w<DQ, NTQ>(dd, i >> 1, u, 2 * (i & 1));   // i = 2 mt + rho
      }
    }
    __syncwarp();
    // the K slot is free (codes consumed, aux read in phase A): request the next chunk's K record
    if (lane == 0 && more) { mbar_expect_tx(&ws.fullk, RB); bulk_g2s(ws.krec, krec + (size_t)(4 * (it + 1)) * RB, RB, &ws.fullk); }
    // ---- D3 (scales) + D4: logits of this thread's 16 tokens x HPW columns, maximum over the chunk -----------
    float corr[HPW], wch[HPW], zsum[HPW];
#pragma unroll
    for (int u = 0; u < HPW; ++u) {
      const float2 sb = ws.hs[ft + 4 * u];
      float mx = -INFINITY;
#pragma unroll
      for (int mp = 0; mp < 4; ++mp)
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const float2 aux = ws.aux_a[32 * mp + 16 * (i >> 1) + 8 * (i & 1) + fg];
          sraw[mp][u][i] = fmaf(aux.x, fmaf(sraw[mp][u][i], sb.x, sb.y), aux.y);
          mx = fmaxf(mx, sraw[mp][u][i]);
        }
      mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 4));
      mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 8));
      mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 16));
      // The fixed-point probabilities refer to the maximum mx of THIS chunk: a token is dropped only if it lies
      // below the resolution relative to the largest of its 127 neighbours, whatever the context length; the chunk's
      // sums enter the running ones with the weight wch = 2^(mx - m_new).  What is rounded is pt = p s1v (probability times
      // the value row scale): the numerator (codes and zero-point sum) uses the rounded pt, the denominator l the EXACT
      // p = pt / s1v -- a token whose V row is tiny against its neighbours' keeps its probability mass in l (its value
      // contribution is below the resolution by construction); numerator and denominator differ by <= 1/2 unit of the
      // fixed point per token, with random sign.
      const float m_new = fmaxf(mr[u], mx);
      corr[u] = ex2_approx(mr[u] - m_new);
      wch[u] = ex2_approx(mx - m_new);
      mr[u] = m_new;
      float2 lz = make_float2(0.f, 0.f);    // {l, zero-point sum} of this thread's tokens
#pragma unroll
      for (int mp = 0; mp < 4; ++mp) {
        const int jp = BITS == 2 ? mp : (mp & 1);
        const uint32_t mul_p = 1u << (BITS * (NCLS - 1 - jp));
        const uint32_t add_p = 0u - ((uint32_t)MAGIC_I * mul_p);
        uint32_t X[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const float2 ab = ws.aux_b[32 * mp + 16 * (i >> 1) + 8 * (i & 1) + fg];   // {1 / s1v, zv}
          const float pt = ex2_approx(sraw[mp][u][i] - mx);
          const float f = fmaf(pt, PF, MAGIC_F);        // fixed-point pt; its radix-256 digits are the low bytes of f's bits
          const float pr = f - MAGIC_F;                 // PF * (rounded pt), an exact integer
          lz = __ffma2_rn(make_float2(pt, pr), ab, lz);   // l from the exact p = pt / s1v, the zero-point sum from the rounded pt
          X[i] = DP == 4 ? __float_as_uint(f) * mul_p + add_p : __float_as_uint(f);
        }
        // column (h, d) of column h = ft + 4u: n-tile (DP / 2) u + (d >> 1), g' = 2 ft + (d & 1); word (kappa = mp, half = fg >> 2, t' = fg & 3)
        if constexpr (DP == 4) {
          uint32_t Y[4];
          transpose4x4(X, Y);
#pragma unroll
          for (int d = 0; d < 4; ++d)
            ws.bfr[2 * u + (d >> 1)][mp >> 1][b_slot(4 * (2 * ft + (d & 1)) + (fg & 3), mp >> 1)][2 * (mp & 1) + (fg >> 2)] = Y[d];
        } else {
          const uint32_t t0 = prmt(X[0], X[1], 0x5140), t1 = prmt(X[2], X[3], 0x5140);
#pragma unroll
          for (int d = 0; d < 2; ++d)
            ws.bfr[u][mp >> 1][b_slot(4 * (2 * ft + d) + (fg & 3), mp >> 1)][2 * (mp & 1) + (fg >> 2)] = prmt(t0, t1, d ? 0x7632 : 0x5410);
        }
      }
      lz.x += __shfl_xor_sync(0xffffffffu, lz.x, 4);  lz.y += __shfl_xor_sync(0xffffffffu, lz.y, 4);
      lz.x += __shfl_xor_sync(0xffffffffu, lz.x, 8);  lz.y += __shfl_xor_sync(0xffffffffu, lz.y, 8);
      lz.x += __shfl_xor_sync(0xffffffffu, lz.x, 16); lz.y += __shfl_xor_sync(0xffffffffu, lz.y, 16);
      zsum[u] = lz.y * (1.f / PF) * wch[u];
      lp[u] = fmaf(lp[u], corr[u], lz.x * wch[u]);     // (every lane with the same ft holds the warp's l of column ft + 4u)
    }
    __syncwarp();
    // ---- D5: value contraction over the 8 m-tiles (rows = channels), accumulate -----------------------------
    {
      uint4 bf[2][NTP];
#pragma unroll
      for (int hk = 0; hk < 2; ++hk)
#pragma unroll
        for (int nu = 0; nu < NTP; ++nu) bf[hk][nu] = *reinterpret_cast<const uint4*>(&ws.bfr[nu][hk][b_slot(lane, hk)][0]);
#pragma unroll
      for (int mp = 0; mp < 4; ++mp) {
        int32_t dd[2][NTP][4];
        contract_mp<BITS, NTP, NTP, false, DP == 2>(ws.vrec, bf, mp, lane, dd, A.shl_mul);
        const uint2 sv = *reinterpret_cast<const uint2*>(&ws.aux_ch[mp][fg][0]);
        const float2 s01 = __half22float2(*reinterpret_cast<const __half2*>(&sv.x)), s23 = __half22float2(*reinterpret_cast<const __half2*>(&sv.y));
        const float s2v[4] = {s01.x, s01.y, s23.x, s23.y};
#pragma unroll
        for (int u = 0; u < HPW; ++u) {
          const float cw = CLS_INV * (1.f / PF) * wch[u];
#pragma unroll
          for (int i = 0; i < 4; ++i)
            ac[mp][u][i] = fmaf(ac[mp][u][i], corr[u], s2v[i] * fmaf(undigit_w<DP, NTP>(dd, i >> 1, u, 2 * (i & 1)), cw, zsum[u]));
        }
      }
    }
    __syncwarp();
    // the V slot is free: request the next chunk's V record
    if (lane == 0 && more) { mbar_expect_tx(&ws.fullv, RB); bulk_g2s(ws.vrec, vrec + (size_t)(4 * (it + 1)) * RB, RB, &ws.fullv); }
  }

  // ---- merge of the 4 private states; hand over to the per-channel layout: thread tid = channel tid -----------
  // every warp stages into ITS OWN dead record slots (no other warp touches them), so no barrier is needed before
  float* stage = reinterpret_cast<float*>(ws.krec);   // [GP][128] floats
  static_assert(RB >= GP * 128 * sizeof(float), "staging area");
#pragma unroll
  for (int u = 0; u < HPW; ++u) {
    if (fg == 0) { sm.wz[warp][ft + 4 * u] = lp[u]; sm.wmax[warp][ft + 4 * u] = mr[u]; }
#pragma unroll
    for (int mp = 0; mp < 4; ++mp)
#pragma unroll
      for (int i = 0; i < 4; ++i) stage[(ft + 4 * u) * 128 + 32 * mp + 16 * (i >> 1) + 8 * (i & 1) + fg] = ac[mp][u][i];
  }
  __syncthreads();
  float m_run[GP], l_part[GP], l_tot[GP], acc[GP];
#pragma unroll
  for (int h = 0; h < GP; ++h) {
    const float m0 = sm.wmax[0][h], m1 = sm.wmax[1][h], m2 = sm.wmax[2][h], m3 = sm.wmax[3][h];
    const float M = fmaxf(fmaxf(m0, m1), fmaxf(m2, m3));
    const float e0 = m0 == -INFINITY ? 0.f : ex2_approx(m0 - M), e1 = m1 == -INFINITY ? 0.f : ex2_approx(m1 - M);
    const float e2 = m2 == -INFINITY ? 0.f : ex2_approx(m2 - M), e3 = m3 == -INFINITY ? 0.f : ex2_approx(m3 - M);
    m_run[h] = M;
    l_tot[h] = fmaf(e0, sm.wz[0][h], fmaf(e1, sm.wz[1][h], fmaf(e2, sm.wz[2][h], e3 * sm.wz[3][h])));
    l_part[h] = tid == 0 ? l_tot[h] : 0.f;
    const float a0 = reinterpret_cast<const float*>(sm.w[0].krec)[h * 128 + tid], a1 = reinterpret_cast<const float*>(sm.w[1].krec)[h * 128 + tid];
    const float a2 = reinterpret_cast<const float*>(sm.w[2].krec)[h * 128 + tid], a3 = reinterpret_cast<const float*>(sm.w[3].krec)[h * 128 + tid];
    acc[h] = fmaf(e0, a0, fmaf(e1, a1, fmaf(e2, a2, e3 * a3)));
  }
  __syncthreads();   // the staged partials are consumed: the slots may now receive the peers' partials, wmax / wz are free
  if (A.cluster > 1) cluster_arrive();
  // dead slots: [0, 16 x WS_STRIDE floats) landing area of the peers' partials, w[2] un-rotated q of the raw windows, w[3] merge weights
  static_assert(sizeof(WS) * 2 >= 16 * WS_STRIDE * sizeof(float) && sizeof(WS) >= GP * 128 * sizeof(float), "landing / scratch areas");
  float* qraw = reinterpret_cast<float*>(&sm.w[2]);
  if (w0.n_sink_tok > 0 || w0.resid > 0 || A.k_blk != nullptr) {   // CTA-uniform: this CTA may run a slice of a raw window
    for (int hh = warp; hh < GP; hh += 4) {
      float v[4] = {0.f, 0.f, 0.f, 0.f};
      if (hh < cm0.ncols) {
        const size_t row = ((size_t)w0.b * cm0.n_q + cm0.tok0 + (hh >> cm0.lg)) * A.Hq + w0.hkv * g + (hh - ((hh >> cm0.lg) << cm0.lg));
        const InT* qp = reinterpret_cast<const InT*>(A.q) + row * D + 4 * lane;
#pragma unroll
        for (int j = 0; j < 4; ++j) v[j] = ld_in<InT>(qp + j) * A.q_scale;
      }
      *reinterpret_cast<float4*>(&qraw[hh * 128 + 4 * lane]) = make_float4(v[0], v[1], v[2], v[3]);
    }
    __syncthreads();
  }
  decode_finish<GP, InT>(A, sm, reinterpret_cast<float*>(&sm.w[0]), reinterpret_cast<float*>(&sm.w[3]), qraw, w0, cm0,
                         do_resid, do_sink, m_run, l_part, l_tot, acc);
}

// LSE merge of R partial sets (e.g. all-gathered from R context-parallel ranks): one CTA per
// (b, q head) row, thread = channel.  parts [R][n_rows][PART_STRIDE]; m is in log2 units of the scaled logits.
__global__ void __launch_bounds__(128) merge_partials_kernel(const float* __restrict__ parts, int R, long long n_rows,
                                                             void* __restrict__ out, int out_dtype) {
  const long long row = blockIdx.x;
  const int tid = threadIdx.x;
  float mstar = -INFINITY;
  for (int r = 0; r < R; ++r) mstar = fmaxf(mstar, parts[((long long)r * n_rows + row) * PART_STRIDE]);
  float L = 0.f, o = 0.f;
  for (int r = 0; r < R; ++r) {
    const float* pr = parts + ((long long)r * n_rows + row) * PART_STRIDE;
    const float w = (pr[0] == -INFINITY) ? 0.f : exp2f(pr[0] - mstar);
    L = fmaf(w, pr[1], L);
    o = fmaf(w, pr[4 + tid], o);
  }
  const float res = L > 0.f ? o / L : 0.f;
  if (out_dtype == KVARN_F32) reinterpret_cast<float*>(out)[row * D + tid] = res;
  else reinterpret_cast<__nv_bfloat16*>(out)[row * D + tid] = __float2bfloat16_rn(res);
}

}  // namespace kvarn

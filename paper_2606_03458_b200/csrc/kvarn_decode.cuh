// kvarn_decode_attention for sm_100a: split-K over 128-token chunks; records staged
// by TMA bulk copies into a shared-memory ring; the two g x 128 x 128 contractions of
// every chunk run on the tensor cores as integer MMAs straight on the packed codes;
// split partials merge through distributed shared memory inside a thread-block cluster.
// SURVEY 8(a) rows D1-D7; DESIGN.md "Decode kernel".
//
//   D1  q' = (q H / sqrt(128)) * sm_scale * log2(e)                    (online Q transform)
//   D2  record (codes + aux) -> shared memory ring, cp.async.bulk + mbarrier
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
// The only rounding is the fixed-point conversion of qt (22 bits + sign relative
// to max_c |qt[h,c]|) and pt (22 bits, pt <= 1); beta and the zero-point term of V
// use the same fixed-point values, so no cancellation error appears between the
// code term and the zero-point term.
//
// Why warp-level mma.sync (IMMA m16n8k32) and not tcgen05: the contraction is tiny
// (N = 4 digits x g heads <= 32 columns) and the kernel is bound by instruction
// issue and by the dependent chain of one chunk, not by tensor throughput.  The
// tcgen05 version of this kernel (git history, profiles/r01b_*) paid two
// TMEM-store -> MMA -> commit -> mbarrier -> TMEM-load round trips and a
// single-thread issue path per chunk; register-level MMAs need 128 (g<=4) or 256
// (g<=8) IMMA per chunk = 270 / 540 tensor-pipe cycles per SM (measured 2.1
// clk/IMMA/SM), below the HBM time of a chunk, with no asynchronous-proxy hand-off.
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

// D (s32, 16x8) += A (u8, 16x32, row) * B (s8 or u8, 32x8, col)
template <bool B_SIGNED>
__device__ __forceinline__ void imma_16832(int32_t (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  if (B_SIGNED)
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

// NCH = chunks processed per loop iteration (per barrier interval).  NCH = 2 gives every warp two
// independent instruction streams between barriers (the kernel is bound by dependent-issue latency,
// not by occupancy: DESIGN.md 6.2) and halves the barriers per chunk.
template <int BITS, int GP, int NCH>
struct DecSmem {
  static constexpr int RB = record_bytes(BITS);
  static constexpr int STAGES = 2;
  static constexpr int NT = GP / 2;            // n-tiles (8 columns each): 4 radix-256 digits x GP heads
  alignas(128) uint8_t rec[STAGES][NCH][2][RB];   // [stage][chunk of the iteration][K | V] records
  // B operands in fragment order: word (nu, kappa, half, lane' = 4 g' + t') -> [nu][hk = kappa>>1][b_slot(lane', hk)][2 (kappa&1) + half]
  alignas(16) uint32_t bq[NCH][NT][2][32][4];
  alignas(16) uint32_t bp[NCH][NT][2][32][4];
  alignas(16) float2 aux_a[NCH][128];          // per MMA row slot of the K tile: {s2, log2 s1v} of its token
  alignas(16) float2 aux_b[NCH][128];          //                                 {1 / s1v, zv}
  alignas(16) float aux_ch[2][NCH][128];       // per channel: s2v / P_FIX (double-buffered by iteration parity)
  alignas(16) float qrot[GP][128];             // q' (rotated, scaled); later: staging of acc / merged acc_rot
  alignas(16) float qraw[GP][128];             // q * q_scale (un-rotated, for the residual window); later p of the residual
  alignas(16) float hs[NCH][GP][2];            // per head: {scale, beta} of the current chunks
  alignas(16) float hmax[GP][4];               // per head: per-warp maxima (over the chunks of the iteration)
  alignas(16) float hz[NCH][GP][4];            // per head: per-warp zero-point sums / l sums
  alignas(16) float wmax[4][GP];               // residual window: per-warp maxima
  alignas(16) float wz[4][GP];                 // residual window / final l: per-warp sums
  alignas(8) uint64_t fullk[STAGES];
  alignas(8) uint64_t fullv[STAGES];
  int last_flag;
};

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

// D[mt][nu] = sum over the 128 K positions of codes (A) x digit planes (B fragments in shared memory);
// the 2 x NT accumulator chains are interleaved so that no IMMA waits for the previous one
template <int BITS, int NT, bool B_SIGNED>
__device__ __forceinline__ void contract(const uint8_t* codes, const uint32_t (*bsm)[2][32][4], int warp, int lane,
                                         int32_t (&d)[2][NT][4]) {
  uint32_t W[2][2][BITS == 2 ? 2 : 4];
  load_row_words<BITS>(codes, warp, lane, 0, W[0]);
  load_row_words<BITS>(codes, warp, lane, 1, W[1]);
#pragma unroll
  for (int mt = 0; mt < 2; ++mt)
#pragma unroll
    for (int nu = 0; nu < NT; ++nu)
#pragma unroll
      for (int c = 0; c < 4; ++c) d[mt][nu][c] = 0;
#pragma unroll
  for (int hk = 0; hk < 2; ++hk) {
    uint4 bf[NT];
#pragma unroll
    for (int nu = 0; nu < NT; ++nu) bf[nu] = *reinterpret_cast<const uint4*>(&bsm[nu][hk][b_slot(lane, hk)][0]);
#pragma unroll
    for (int k1 = 0; k1 < 2; ++k1) {
      const int kappa = 2 * hk + k1;
      uint32_t a[2][4];
      a_frag<BITS>(W[0], kappa, a[0]);
      a_frag<BITS>(W[1], kappa, a[1]);
#pragma unroll
      for (int nu = 0; nu < NT; ++nu)
#pragma unroll
        for (int mt = 0; mt < 2; ++mt) {
          if (k1) imma_16832<B_SIGNED>(d[mt][nu], a[mt], bf[nu].z, bf[nu].w);
          else imma_16832<B_SIGNED>(d[mt][nu], a[mt], bf[nu].x, bf[nu].y);
        }
    }
  }
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

template <int BITS, int GP, int NCH, typename InT>
#ifndef KVARN_DEC_OCC4
#define KVARN_DEC_OCC4 4
#endif
#ifndef KVARN_DEC_OCC8
#define KVARN_DEC_OCC8 4
#endif
// GP = 4: four resident CTAs per SM with either NCH (128 registers; the two-chunk variant's 55.6 KB of shared memory
// fits four times in 228 KB) -- with three, the 64k-context case drops from 195 to 213 us
__global__ void __launch_bounds__(128, GP == 4 ? KVARN_DEC_OCC4 : KVARN_DEC_OCC8 / NCH) decode_kernel(const DecodeArgs A) {
  using SM = DecSmem<BITS, GP, NCH>;
  constexpr int RB = SM::RB, STAGES = SM::STAGES, NT = SM::NT;
  constexpr int NCLS = 8 / BITS;
  constexpr float CLS_INV = BITS == 2 ? (1.f / 64.f) : (1.f / 16.f);  // 1 / CLSMAX
  constexpr int HPW = GP / 4;   // heads per warp in the B_q builder = heads per thread in the softmax (h = t + 4u)

  extern __shared__ __align__(128) uint8_t smem_raw[];
  SM& sm = *reinterpret_cast<SM*>(smem_raw);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int fg = lane >> 2, ft = lane & 3;   // MMA fragment coordinates: row group g, thread-in-group t
  const int g = A.g;
  float mr[HPW], lp[HPW], ac[HPW][4];   // running maximum, partial l, partial accumulator of this thread's (heads, rows)
  const Where w0 = where_am_i<false>(A);
  const ColMap cm0 = col_map<false>(A);   // before the main loop: q rows of D1, block weight of the split plan
  const bool do_resid0 = (w0.split == A.splits - 1) && w0.resid > 0;
  const bool do_sink0 = (w0.split == 0) && w0.n_sink_tok > 0;
  {   // ======== setup + main loop: everything declared here dies before the epilogue ========
  const int bh = w0.bh, b = w0.b, hkv = w0.hkv, split = w0.split;

  // ---- chunk range of this split ----------------------------------------------------
  const int n_sink_tok = w0.n_sink_tok, n_chunks = w0.n_chunks, resid = w0.resid;
  // Balanced split: a raw window (512 B per token against 72 B) weighs like one chunk per 12 tokens (measured:
  // 127 residual tokens cost a CTA about 10 chunks), so the splits that own the sink / residual window get
  // correspondingly fewer chunks.  Virtual units: [sink | chunk 0 .. n_chunks-1 | residual].
  const int w_sink = (n_sink_tok + 11) / 12, w_res = (resid + cm0.blk_cnt + 11) / 12;
  const int per = (n_chunks + w_sink + w_res + A.splits - 1) / A.splits;
  const int c_begin = min(max(split * per - w_sink, 0), n_chunks);
  const int c_end = min(max((split + 1) * per - w_sink, 0), n_chunks);
  const int n_my = c_end - c_begin;

  const uint8_t* krec = A.k_records + ((size_t)bh * A.max_chunks + c_begin) * RB;
  const uint8_t* vrec = A.v_records + ((size_t)bh * A.max_chunks + c_begin) * RB;

  // ---- setup: barriers, first TMA loads, q ------------------------------------------
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < STAGES; ++s) { mbar_init(&sm.fullk[s], 1); mbar_init(&sm.fullv[s], 1); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
#pragma unroll
    for (int s = 0; s < STAGES; ++s) {
      const int nc = min(NCH, n_my - s * NCH);   // chunks of iteration s
      if (nc > 0) {
        mbar_expect_tx(&sm.fullk[s], nc * RB);
        mbar_expect_tx(&sm.fullv[s], nc * RB);
        for (int c = 0; c < nc; ++c) {
          bulk_g2s(sm.rec[s][c][0], krec + (size_t)(s * NCH + c) * RB, RB, &sm.fullk[s]);
          bulk_g2s(sm.rec[s][c][1], vrec + (size_t)(s * NCH + c) * RB, RB, &sm.fullv[s]);
        }
      }
    }
  }

  // D1: q' = (q H / sqrt(128)) * q_scale; heads >= g are zero
  for (int hh = warp; hh < GP; hh += 4) {
    float v[4] = {0.f, 0.f, 0.f, 0.f};
    if (hh < cm0.ncols) {
      const size_t row = ((size_t)b * cm0.n_q + cm0.tok0 + (hh >> cm0.lg)) * A.Hq + hkv * g + (hh - ((hh >> cm0.lg) << cm0.lg));
      const InT* qp = reinterpret_cast<const InT*>(A.q) + row * D + 4 * lane;
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
  __syncthreads();

  // B_q builder role: warp -> heads warp (+4); lane = 8 kappa + 4 half + t' owns the four K positions
  // p = 16 half + 4 t' + b (b = 0..3) of k-step kappa, i.e. one 32-bit word of a B fragment per digit
  const int bk = lane >> 3, bhalf = (lane >> 2) & 1, btp = lane & 3;
  float qreg[HPW][4];
#pragma unroll
  for (int bb = 0; bb < 4; ++bb) {
    const int ch = BITS == 2 ? 16 * btp + 4 * bb + bk + 64 * bhalf
                             : 8 * (btp + 4 * (2 * (bk >> 1) + bhalf)) + 2 * bb + (bk & 1);
#pragma unroll
    for (int u = 0; u < HPW; ++u) qreg[u][bb] = sm.qrot[warp + 4 * u][ch];
  }
  // fixed-point value -> digits: X = (bits(f) - MAGIC_I) << shift, balanced:  (X + 0x80808080) ^ 0x80808080
  const int jq = BITS == 2 ? bk : (bk & 1);
  const uint32_t mul_q = 1u << (BITS * (NCLS - 1 - jq));
  const uint32_t add_q = 0x80808080u - ((uint32_t)MAGIC_I * mul_q);
  // column (h, d) of head h = warp + 4u: n-tile 2u + (d >> 1), g' = 2 warp + (d & 1); lane' = 4 g' + t'
  uint32_t* bq_dst[2];
#pragma unroll
  for (int dd = 0; dd < 2; ++dd) bq_dst[dd] = &sm.bq[0][0][bk >> 1][b_slot(4 * (2 * warp + dd) + btp, bk >> 1)][2 * (bk & 1) + bhalf];
  // softmax role: thread (warp, fg, ft) sees tokens slot(mt, rho) = 32 warp + 16 mt + 8 rho + fg, heads ft + 4u;
  // these four tokens are K positions b = 2 mt + rho of word (kappa = warp, half = fg >> 2, t' = fg & 3)
  const int jp = BITS == 2 ? warp : (warp & 1);
  const uint32_t mul_p = 1u << (BITS * (NCLS - 1 - jp));
  const uint32_t add_p = 0u - ((uint32_t)MAGIC_I * mul_p);
  // column (h, d) of head h = ft + 4u: n-tile 2u + (d >> 1), g' = 2 ft + (d & 1); lane' = 4 g' + t'
  uint32_t* bp_dst[2];
#pragma unroll
  for (int dd = 0; dd < 2; ++dd) bp_dst[dd] = &sm.bp[0][0][warp >> 1][b_slot(4 * (2 * ft + dd) + (fg & 3), warp >> 1)][2 * (warp & 1) + (fg >> 2)];
  constexpr int B_CH = NT * 256;   // 32-bit words of one chunk's B operand

#pragma unroll
  for (int u = 0; u < HPW; ++u) {
    mr[u] = -INFINITY; lp[u] = 0.f;
#pragma unroll
    for (int i = 0; i < 4; ++i) ac[u][i] = 0.f;
  }

  // One loop iteration = NCH chunks.  FULL (all NCH chunks present) is a compile-time flag so that the
  // common case has no per-chunk branches and the chunks' instruction streams interleave.
  auto iteration = [&](auto full_tag, const int it) {
    constexpr bool FULL = decltype(full_tag)::value;
    const int st = it % STAGES;
    const uint32_t par = (it / STAGES) & 1;
    const int nc = min(NCH, n_my - it * NCH);   // chunks of this iteration (uniform)
    mbar_wait(&sm.fullk[st], par);

    // ---- phase A: B_q (digits of the fixed-point qt), beta, per-token / per-channel aux -----------
#pragma unroll
    for (int c = 0; c < NCH; ++c) {
      if (FULL || c < nc) {
        const uint8_t* kr = sm.rec[st][c][0];
        // aux of the K record in builder order: s1[4 lane + b], z[4 lane + b]
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
          const float inv = amax[u] > 1e-30f ? Q_FIX * rcp_approx(amax[u]) : 0.f;
          uint32_t X[4], Y[4];
#pragma unroll
          for (int r = 0; r < 4; ++r) {
            const float f = fmaf(qt[u][r], inv, MAGIC_F);            // integer Q in the low mantissa bits
            X[r] = (__float_as_uint(f) * mul_q + add_q) ^ 0x80808080u;   // balanced s8 digits of Q << shift
          }
          transpose4x4(X, Y);   // Y[d] = digit d of the four K positions = one B-fragment word of column (h, d)
#pragma unroll
          for (int d = 0; d < 4; ++d) bq_dst[d & 1][c * B_CH + (2 * u + (d >> 1)) * 256] = Y[d];
          if (lane == 0) {
            const float sc = amax[u] * (1.f / Q_FIX);
            sm.hs[c][h][0] = sc * CLS_INV;   // logit = s2 * (acc * scale + beta)
            sm.hs[c][h][1] = bsum[u];
          }
        }
      }
    }
    mbar_wait(&sm.fullv[st], par);
#pragma unroll
    for (int c = 0; c < NCH; ++c) {
      if (FULL || c < nc) {
        // thread tid: aux of MMA row slot tid of the K tile (token-indexed arrays are stored in slot order)
        // and of channel tid of the V tile
        const uint8_t* kr = sm.rec[st][c][0];
        const uint8_t* vr = sm.rec[st][c][1];
        const float s2t = e4m3_to_f32(kr[s2_off(BITS) + tid]);
        const float s1v = fmaxf(e4m3_to_f32(vr[s1_off(BITS) + tid]), 9.094947e-13f);   // 2^-40: a zero scale stays harmless
        const float zv = f16_bits_to_f32(reinterpret_cast<const uint16_t*>(vr + z_off(BITS))[tid]);
        // pt = p s1v = exp2(logit + log2 s1v - m): the running maximum is taken over the shifted logits,
        // so pt <= 1 and its fixed-point scale is a constant
        sm.aux_a[c][tid] = make_float2(s2t, lg2_approx(s1v));
        sm.aux_b[c][tid] = make_float2(rcp_approx(s1v) * (1.f / P_FIX), zv);
        sm.aux_ch[it & 1][c][tid] = e4m3_to_f32(vr[s2_off(BITS) + tid]) * (1.f / P_FIX);
      }
    }
    __syncthreads();                                                   // barrier 1
    // every warp is done with iteration it-1: refill its V slots (its K slots were refilled after barrier 2)
    if (tid == 0 && it >= 1) {
      const int nxt = it - 1 + STAGES, s2 = (it - 1) % STAGES;
      const int nn = min(NCH, n_my - nxt * NCH);
      if (nn > 0) {
        mbar_expect_tx(&sm.fullv[s2], nn * RB);
        for (int c = 0; c < nn; ++c) bulk_g2s(sm.rec[s2][c][1], vrec + (size_t)(nxt * NCH + c) * RB, RB, &sm.fullv[s2]);
      }
    }

    // ---- D3: logits of this thread's 4 tokens x HPW heads (per chunk) -----------------------------------
    float logit[NCH][HPW][4];
#pragma unroll
    for (int c = 0; c < NCH; ++c) {
      if (FULL || c < nc) {
        int32_t dd[2][NT][4];
        contract<BITS, NT, true>(sm.rec[st][c][0], sm.bq[c], warp, lane, dd);
        float2 aux[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) aux[i] = sm.aux_a[c][32 * warp + 16 * (i >> 1) + 8 * (i & 1) + fg];
#pragma unroll
        for (int u = 0; u < HPW; ++u) {
          const float2 sb = *reinterpret_cast<const float2*>(sm.hs[c][ft + 4 * u]);
#pragma unroll
          for (int i = 0; i < 4; ++i) {   // i = 2 mt + rho
            const int mt = i >> 1, cc = 2 * (i & 1);
            const float a = undigit(dd[mt][2 * u][cc], dd[mt][2 * u][cc + 1], dd[mt][2 * u + 1][cc], dd[mt][2 * u + 1][cc + 1]);
            logit[c][u][i] = fmaf(aux[i].x, fmaf(a, sb.x, sb.y), aux[i].y);
          }
        }
      } else {
#pragma unroll
        for (int u = 0; u < HPW; ++u)
#pragma unroll
          for (int i = 0; i < 4; ++i) logit[c][u][i] = -INFINITY;
      }
    }
    // ---- D4: online softmax -----------------------------------------------------------------------------
#pragma unroll
    for (int u = 0; u < HPW; ++u) {
      float mx = -INFINITY;
#pragma unroll
      for (int c = 0; c < NCH; ++c)
        mx = fmaxf(mx, fmaxf(fmaxf(logit[c][u][0], logit[c][u][1]), fmaxf(logit[c][u][2], logit[c][u][3])));
      mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 4));
      mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 8));
      mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 16));
      if (fg == 0) sm.hmax[ft + 4 * u][warp] = mx;
    }
    __syncthreads();                                                   // barrier 2
    // every warp is done with the K records of this iteration: prefetch iteration it + STAGES into their slots
    if (tid == 0) {
      const int nxt = it + STAGES;
      const int nn = min(NCH, n_my - nxt * NCH);
      if (nn > 0) {
        mbar_expect_tx(&sm.fullk[st], nn * RB);
        for (int c = 0; c < nn; ++c) bulk_g2s(sm.rec[st][c][0], krec + (size_t)(nxt * NCH + c) * RB, RB, &sm.fullk[st]);
      }
    }
    // The fixed-point probabilities refer to the maximum m_it of THIS iteration's chunks (not to the running
    // maximum): a token is dropped only if it lies 2^-23 below the largest of its own <= 256 neighbours, so the
    // dropped mass is bounded by 255 * 2^-23 whatever the context length; the iteration's sums enter the running
    // ones with the weight wch = 2^(m_it - m_new).  l is accumulated from the SAME rounded values as the
    // numerator, so numerator and denominator stay consistent.
    float corr[HPW], wch[HPW];
#pragma unroll
    for (int u = 0; u < HPW; ++u) {
      const float4 hm = *reinterpret_cast<const float4*>(sm.hmax[ft + 4 * u]);
      const float m_it = fmaxf(fmaxf(hm.x, hm.y), fmaxf(hm.z, hm.w));
      const float m_new = fmaxf(mr[u], m_it);
      corr[u] = ex2_approx(mr[u] - m_new);
      wch[u] = ex2_approx(m_it - m_new);
      mr[u] = m_new;
      float lsum = 0.f;
#pragma unroll
      for (int c = 0; c < NCH; ++c) {
        if (FULL || c < nc) {
          uint32_t X[4], Y[4];
          float zpart = 0.f;
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const float2 ab = sm.aux_b[c][32 * warp + 16 * (i >> 1) + 8 * (i & 1) + fg];   // {1 / (s1v P_FIX), zv}
            const float pt = ex2_approx(logit[c][u][i] - m_it);
            // D5 prep: fixed-point pt; its radix-256 digits are the bytes of X
            const float f = fmaf(pt, P_FIX, MAGIC_F);
            const float pr = f - MAGIC_F;                 // P_FIX * (rounded pt), an exact integer
            lsum = fmaf(pr, ab.x, lsum);
            zpart = fmaf(pr, ab.y, zpart);
            X[i] = __float_as_uint(f) * mul_p + add_p;
          }
          transpose4x4(X, Y);
#pragma unroll
          for (int d = 0; d < 4; ++d) bp_dst[d & 1][c * B_CH + (2 * u + (d >> 1)) * 256] = Y[d];
          zpart += __shfl_xor_sync(0xffffffffu, zpart, 4);
          zpart += __shfl_xor_sync(0xffffffffu, zpart, 8);
          zpart += __shfl_xor_sync(0xffffffffu, zpart, 16);
          if (fg == 0) sm.hz[c][ft + 4 * u][warp] = zpart;
        }
      }
      lp[u] = fmaf(lp[u], corr[u], lsum * wch[u]);
    }
    __syncthreads();                                                   // barrier 3

    // ---- D5: this thread's 4 channels x HPW heads of the value contraction ---------------------------
#pragma unroll
    for (int u = 0; u < HPW; ++u)
#pragma unroll
      for (int i = 0; i < 4; ++i) ac[u][i] *= corr[u];
#pragma unroll
    for (int c = 0; c < NCH; ++c) {
      if (FULL || c < nc) {
        int32_t dd[2][NT][4];
        contract<BITS, NT, false>(sm.rec[st][c][1], sm.bp[c], warp, lane, dd);
        float s2v[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) s2v[i] = sm.aux_ch[it & 1][c][32 * warp + 16 * (i >> 1) + 8 * (i & 1) + fg];
#pragma unroll
        for (int u = 0; u < HPW; ++u) {
          const float4 hz = *reinterpret_cast<const float4*>(sm.hz[c][ft + 4 * u]);
          const float zsum = ((hz.x + hz.y) + (hz.z + hz.w)) * wch[u];
          const float cw = CLS_INV * wch[u];
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int mt = i >> 1, cc = 2 * (i & 1);
            const float a = undigit(dd[mt][2 * u][cc], dd[mt][2 * u][cc + 1], dd[mt][2 * u + 1][cc], dd[mt][2 * u + 1][cc + 1]);
            ac[u][i] = fmaf(s2v[i], fmaf(a, cw, zsum), ac[u][i]);
          }
        }
      }
    }
  };
  const int n_it = (n_my + NCH - 1) / NCH;
  for (int it = 0; it < n_it; ++it) {
    if (NCH == 1 || n_my - it * NCH >= NCH) iteration(std::true_type{}, it);
    else iteration(std::false_type{}, it);
  }
  }   // ======== end of setup + main loop ========

  // ---- hand over to the per-channel layout of the residual window / merge: thread tid = channel tid ----
  __syncthreads();
  // Re-derive the CTA's coordinates / column map instead of carrying them through the loop where that pays
  // (64k context, g = 8: 2-bit 367 -> 344 us, 4-bit 390 -> 350 us); the 2-bit g <= 4 kernel is faster with them
  // live (195 vs 199 us, 203 vs 209 us with a full residual window), so it keeps them.
  const Where w1 = BITS == 4 ? where_am_i<true>(A) : w0;
  const int bh = w1.bh, b = w1.b, hkv = w1.hkv, split = w1.split, n_sink_tok = w1.n_sink_tok, resid = w1.resid;
  const bool do_resid = BITS == 4 ? ((split == A.splits - 1) && resid > 0) : do_resid0;
  const bool do_sink = BITS == 4 ? ((split == 0) && n_sink_tok > 0) : do_sink0;
  const ColMap cm = (GP == 8 || BITS == 4) ? col_map<true>(A) : cm0;
  const int lg = cm.lg, tok0 = cm.tok0, ncols = cm.ncols, n_q = cm.n_q, blk_cnt = cm.blk_cnt;
  const bool has_blk = A.k_blk != nullptr;
  const bool do_blk = (split == A.splits - 1) && has_blk;
  auto qrow = [&](int j) -> size_t { return ((size_t)b * n_q + tok0 + (j >> lg)) * A.Hq + hkv * g + (j - ((j >> lg) << lg)); };
  // every warp has left the main loop and no TMA fill is outstanding: this CTA's record ring is dead and may
  // receive the peers' partials.  Arrive now, wait only right before the first DSMEM store (D7a), so the
  // barrier latency hides behind the raw windows and the l reductions.
  if (A.cluster > 1) cluster_arrive();
#pragma unroll
  for (int u = 0; u < HPW; ++u) {
    float l = lp[u];
    l += __shfl_xor_sync(0xffffffffu, l, 4);
    l += __shfl_xor_sync(0xffffffffu, l, 8);
    l += __shfl_xor_sync(0xffffffffu, l, 16);
    if (fg == 0) { sm.hz[0][ft + 4 * u][warp] = l; if (warp == 0) sm.hs[0][ft + 4 * u][0] = mr[u]; }
#pragma unroll
    for (int i = 0; i < 4; ++i) sm.qrot[ft + 4 * u][32 * warp + 16 * (i >> 1) + 8 * (i & 1) + fg] = ac[u][i];
  }
  __syncthreads();
  float m_run[GP], l_part[GP], l_tot[GP], acc[GP];
#pragma unroll
  for (int h = 0; h < GP; ++h) {
    m_run[h] = sm.hs[0][h][0];
    const float4 hz = *reinterpret_cast<const float4*>(sm.hz[0][h]);
    l_tot[h] = (hz.x + hz.y) + (hz.z + hz.w);                     // l of the chunks (every thread has it)
    l_part[h] = tid == 0 ? l_tot[h] : 0.f;                        // with raw windows: thread 0 carries it into the sum
    acc[h] = sm.qrot[h][tid];
  }

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
            const float4 q0 = *reinterpret_cast<const float4*>(&sm.qraw[h][c]);
            const float4 q1 = *reinterpret_cast<const float4*>(&sm.qraw[h][c + 4]);
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
      const float corr = exp2f(m_run[h] - m_new);
      m_run[h] = m_new;
      p[h] = exp2f(logit[h] - m_new);        // exp2(-inf) = 0 for masked tokens
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
  if (do_sink)
    raw_window(reinterpret_cast<const InT*>(A.k_sink) + (size_t)bh * A.n_sink * D,
               reinterpret_cast<const InT*>(A.v_sink) + (size_t)bh * A.n_sink * D, n_sink_tok, NO_MASK);
  if (do_resid)
    raw_window(reinterpret_cast<const InT*>(A.k_resid) + (size_t)bh * G * D,
               reinterpret_cast<const InT*>(A.v_resid) + (size_t)bh * G * D, resid, NO_MASK);
  if (do_blk)
    raw_window(reinterpret_cast<const InT*>(A.k_blk) + (size_t)bh * n_q * D,
               reinterpret_cast<const InT*>(A.v_blk) + (size_t)bh * n_q * D, blk_cnt, tok0);

  // ---- l: reduce the per-thread partial sums (only a CTA that ran a raw window has any beyond the chunks') ----
  if (do_sink || do_resid || do_blk) {   // CTA-uniform
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
    float* land = reinterpret_cast<float*>(&sm.rec[0][0][0]);   // [<= 16][WS_STRIDE]
    static_assert(sizeof(sm.rec) >= 16 * WS_STRIDE * sizeof(float), "landing area");
    cluster_wait();
    const uint32_t land_addr = smem_u32(land);
#pragma unroll
    for (int h = 0; h < GP; ++h) {
      if (h < ncols) {
        const int j = h / CS, d = h - j * CS;
        const uint32_t dst = mapa_shared(land_addr + (uint32_t)(j * CS + crank) * (WS_STRIDE * 4), (uint32_t)d);
        if (tid == 0) { st_cluster_f32(dst, m_run[h]); st_cluster_f32(dst + 4, l_tot[h]); }
        st_cluster_f32(dst + 16 + 4 * tid, acc[h]);
        if (do_resid || do_sink || do_blk) st_cluster_f32(dst + 16 + 512 + 4 * tid, acc_res[h]);
      }
    }
    cluster_sync_all();
    const bool res_here = (resid > 0 || has_blk) && split / CS == NC - 1;   // this cluster's last rank ran the residual window
    const bool sink_here = n_sink_tok > 0 && split / CS == 0;    // this cluster's rank 0 ran the sink window
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
          if ((res_here && r == CS - 1) || (sink_here && r == 0)) rj = fmaf(w, sl[132 + tid], rj);
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
    float* wsp = reinterpret_cast<float*>(sm.bq);   // [GP][64] weights (B_q is dead by now)
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
    sm.qraw[j][tid] = (l_tot[j] > 0.f) ? acc_res[j] : 0.f;
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
    const float4 s4 = *reinterpret_cast<const float4*>(&sm.qraw[jj][4 * lane]);
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

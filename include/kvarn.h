/*
 * kvarn.h -- C ABI of the KVarN hot path for NVIDIA B200 (sm_100a).
 *
 * KVarN (arxiv/paper_2606_03458; cited as P:<line> of PAPER.md) compresses the
 * KV cache tile by tile: every (head_dim=128 x 128-token) tile of one KV head
 * is Hadamard-rotated along head_dim (Fig. 2), variance-normalised
 * along both axes by Algorithm 1 "VarN", quantised by
 * asymmetric round-to-nearest -- K per channel, V per token, Eq. 1 --
 * and stored as packed 2-bit (or 4-bit) codes plus, per 128 elements, two FP8
 * scales and one FP16 zero-point = 2.25 bit/element.  Decoding reads
 * that cache directly (P:9): kvarn_decode_attention computes
 * softmax(q K^T * sm_scale) V over [dequantised chunks ; raw residual tokens]
 * without ever materialising a dequantised cache.
 *
 * Entry points: kvarn_quantize_chunk / kvarn_prefill (bulk write path), kvarn_append / kvarn_append_block
 * (on-the-fly compression while decoding), kvarn_decode_attention (read path), kvarn_block_attention /
 * kvarn_block_attention_dense (a block of new tokens against the cache, Fig. 4),
 * kvarn_decode_attention_partial + kvarn_merge_partials (a sequence spread over several caches / GPUs),
 * kvarn_decode_attention_static (the read path with its scratch inside the library: allocates nothing),
 * kvarn_rope_hadamard / kvarn_hadamard_rows / kvarn_hadamard_row_groups (the Hadamard arrangement of App. A), the *_host forms, layout queries and the record pack / unpack test hooks.
 *
 * Conventions
 *   - "DEVICE" pointers are CUDA device memory owned by the caller; "HOST"
 *     pointers are ordinary (preferably pinned) host memory.  The library
 *     allocates no device memory, keeps no global state (one exception: the static
 *     scratch array of kvarn_decode_attention_static) and never synchronises
 *     the device: every call only enqueues work on the caller's `stream`
 *     (a cudaStream_t passed as void*; NULL = the legacy default stream).
 *   - All calls return a kvarn_status (0 = OK, negative = error); nothing is
 *     enqueued when a negative status is returned.  No C++ exception crosses
 *     this boundary.  Non-finite inputs give undefined codes but never fault.
 *   - A "tile" is 128 tokens x 128 channels of ONE KV head, row-major
 *     [token][channel], of K or of V.  A "record" is the stored form of one
 *     tile; its internal packing is opaque (use kvarn_unpack_record_host).
 */
#ifndef KVARN_H_
#define KVARN_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define KVARN_API __attribute__((visibility("default")))
#else
#define KVARN_API
#endif

#define KVARN_HEAD_DIM 128
#define KVARN_CHUNK 128
#define KVARN_MAX_ITERS 16

typedef enum {
  KVARN_OK = 0,
  KVARN_INVALID_ARG = -1,         /* null pointer, non-positive size, Hq % Hkv != 0 */
  KVARN_UNSUPPORTED = -2,         /* head_dim/chunk != 128, bits not in {2,4}, g not in 1..8, dtype */
  KVARN_MISALIGNED = -3,          /* a pointer or stride is not 16-byte aligned */
  KVARN_WORKSPACE_TOO_SMALL = -4, /* ws_bytes < kvarn_decode_workspace_bytes(...) */
  KVARN_CAPACITY = -5,            /* host-checkable capacity bound violated */
  KVARN_CUDA = -6                 /* cudaGetLastError() after a launch / copy was not cudaSuccess */
} kvarn_status;

typedef enum { KVARN_BF16 = 0, KVARN_F32 = 1 } kvarn_dtype;
typedef enum { KVARN_KIND_K = 0, KVARN_KIND_V = 1 } kvarn_kind;

/* Method parameters (POD, caller-filled; kvarn_default_params gives the paper's). */
typedef struct {
  int32_t head_dim;  /* must be 128 */
  int32_t chunk;     /* tokens per quantisation group G; must be 128 */
  int32_t bits;      /* 2 (paper) or 4 */
  int32_t iters;     /* Algorithm 1's K; 8 in Sec. 4.2; 0..KVARN_MAX_ITERS */
  float var_min;     /* c_min of Alg. 1: lower clamp on variances; default 1e-8 */
  float var_max;     /* c_max of Alg. 1; default 1e8 */
  float log_lo;      /* lower clamp of the log-scales, -0.3 */
  float log_hi;      /* upper clamp of the log-scales, 10.0 */
  int32_t rotate_k;  /* 1: Hadamard-rotate K tiles (and q inside decode) */
  int32_t rotate_v;  /* 1: Hadamard-rotate V tiles (and un-rotate the output) */
  int32_t in_dtype;  /* kvarn_dtype of K, V, q and of the residual window */
  int32_t out_dtype; /* kvarn_dtype of the attention output */
  int32_t splits;    /* decode split-K factor over chunks; 0 = choose automatically.  A value s > 0 runs
                      * c = the largest divisor of s that is <= 8 CTAs per thread-block cluster (merged
                      * through distributed shared memory) and s / c clusters merged through the workspace */
  int32_t aux_round; /* 0 (default): codes from the unrounded scale / zero-point, aux rounded to FP8 / FP16 for
                      * storage afterwards.  1 ("round-before"): the second scale is rounded to FP8 before the
                      * tile is balanced and RTN runs against the STORED step s1 / absorbed scale and the
                      * stored FP16 zero-point, so the FP8 error of the scales is absorbed by the codes
                      * (P:382 does not say which; at 4-bit it cuts the token-magnitude error ~3x). */
  int32_t decode_digits; /* precision of the decode kernel's integer tensor-core operands.  0 (default): q~ 22-bit, p~ 16-bit
                      * fixed point (four / two radix-256 digit planes); 2 (2-bit caches): q~ 15 bits + sign, p~ 16 bits
                      * (half the tensor-core work; error up to ~1e-3 of the 2e-3 tolerance on short, peaked contexts);
                      * 4: 22 / 22 bits. */
} kvarn_params;

/* Byte layout of one record (fixed by bits): codes | s1[128] e4m3 | s2[128] e4m3 | z[128] f16.
 * codes: K records hold one row per TOKEN (its 128 channels), V records one row
 * per CHANNEL (its 128 tokens); a row is little-endian (element e at bit
 * bits*(e % (8/bits)) of byte e*bits/8).  Rows are the M rows of the decode
 * kernel's integer MMAs (m16n8k32): row slot s = 32*warp + 16*mtile + 8*rho + g
 * is held by the threads (g = lane>>2, t = lane&3) of `warp`, and thread t
 * expands the 32-bit words t, t+4 (, t+8, t+12 at 4-bit) of the row.  Byte b of
 * word wi = 4*q + t of slot s sits at
 *     2-bit: warp*1024 + mtile*512 + (4*g + t)*16 + rho*8 + q*4 + b
 *     4-bit: warp*2048 + mtile*1024 + rho*512 + (4*g + t)*16 + q*4 + b
 * (one conflict-free 16-byte shared-memory load per lane).  In the contraction
 * element e of a row is position p of k-step kappa:
 *     2-bit: kappa = e & 3,               p = 16*(e>>6) + 4*((e>>4)&3) + ((e>>2)&3)
 *     4-bit: kappa = 2*(e>>6) + (e&1),    p = 16*((e>>5)&1) + 4*((e>>3)&3) + ((e>>1)&3)
 * V rows use slot = channel.  K rows use slot(token tau) = 32*kappa(tau) +
 * 16*(b>>1) + 8*(b&1) + 4*(p>>4) + ((p>>2)&3) with b = p & 3 -- the four tokens
 * a thread sees after the QK^T MMA are then one 32-bit word of the B operand of
 * the value MMA.
 * s1 = FP8-E4M3 absorbed scale of the RTN group (K: per channel, V: per token),
 * s2 = FP8-E4M3 second (Sinkhorn) scale of the other axis, z = FP16 zero-point
 * of the RTN group (Eq. 1: x_dq = (code + z) * s1 * s2).  Per-token
 * arrays (K.s2, V.s1, V.z) are indexed by slot(token); K.s1 and K.z (per
 * channel) by 4*(8*kappa + (p>>2)) + (p&3) of the channel (the order in which
 * the decode kernel's B-operand builder reads them); V.s2 by channel.
 * kvarn_unpack_record_host gives the canonical view (codes[t][c], natural order). */
typedef struct {
  size_t record_bytes; /* 4608 at 2-bit, 8704 at 4-bit (=> 2.25 / 4.25 bit per element) */
  size_t codes_off, codes_bytes;
  size_t s1_off, s2_off, z_off; /* 128 x u8, 128 x u8, 128 x f16 */
} kvarn_layout_info;

/* The cache of one attention layer in the paper's three-region layout: n_sink sink tokens
 * kept in in_dtype ("S sink tokens in FP16", S = 128 or 32 in the paper; 0 = no sink region), the
 * quantised body of 128-token groups, and the trailing not-yet-quantised tokens.  For a sequence of
 * len tokens:  sink = min(len, n_sink),  chunks = max(len - n_sink, 0) / 128,
 * residual = max(len - n_sink, 0) % 128.  All DEVICE pointers. */
typedef struct {
  void* k_records;      /* [B][Hkv][max_chunks][record_bytes], 16-B aligned */
  void* v_records;      /* same shape */
  void* k_resid;        /* [B][Hkv][128][128] in_dtype: raw (un-rotated) residual tokens */
  void* v_resid;        /* same shape */
  int32_t* seq_lens;    /* [B] tokens held per sequence: chunks = len/128, residual = len%128 */
  int32_t* ticket;      /* [B] scratch for kvarn_append, zero-initialised by the caller once */
  int32_t* decode_ticket; /* [B*Hkv] scratch for kvarn_decode_attention (arrival counters of the split-K
                           * merge), zero-initialised by the caller once; every call leaves it zero.
                           * Calls that share it must be ordered on one stream. */
  int32_t B, Hkv, max_chunks;
  int32_t n_sink;       /* S: tokens [0, S) of every sequence stay raw in k_sink / v_sink; 0..128 */
  void* k_sink;         /* [B][Hkv][n_sink][128] in_dtype (may be NULL when n_sink = 0) */
  void* v_sink;         /* same shape */
  /* Capacity of a sequence: n_sink + max_chunks*128 + 127 tokens.  Two optional guards of the append path: */
  int32_t max_len_hint; /* HOST knowledge: an upper bound on max_b seq_lens[b] before the call (the caller counts the
                         * tokens it appends); <= 0 = unknown.  When > 0, kvarn_append / kvarn_append_block return
                         * KVARN_CAPACITY and enqueue nothing if max_len_hint + n_new exceeds the capacity. */
  int32_t* overflow;    /* DEVICE, nullable: sticky counter, incremented once per (sequence, call) whose tokens did
                         * not fit and were dropped (lengths the host cannot bound); never reset by the library. */
} kvarn_cache;

/* Optional per-tile debug outputs of the quantizer (all DEVICE, each nullable).
 * Index [kind][tile] with kind 0 = K, 1 = V.  Values are the fp32 numbers
 * BEFORE FP8/FP16 storage rounding, so tests can compare against the oracle at
 * the iterate the kernel kept (Alg. 1 line 18 is degenerate between iterates
 * whose imbalance agrees to rounding). */
typedef struct {
  int32_t* k_best; /* [2][n_tiles]            iterate kept by the "<=" rule (0..iters) */
  float* imb;      /* [2][n_tiles][KVARN_MAX_ITERS+1] imbalance I_k, k = 0..iters */
  float* aux_f32;  /* [2][n_tiles][3][128]    s1, s2, z as fp32 (indexing as in the record) */
} kvarn_debug;

KVARN_API void kvarn_default_params(kvarn_params* p, int32_t bits);
KVARN_API const char* kvarn_status_string(int status);
KVARN_API int kvarn_version(void);

/* Record layout for p->bits.  Returns KVARN_UNSUPPORTED for other bit widths. */
KVARN_API int kvarn_layout(const kvarn_params* p, kvarn_layout_info* out);

/* Bytes of DEVICE workspace kvarn_decode_attention needs for this shape (partials of the
 * cross-cluster merge; touched only when more than one cluster shares a sequence). */
KVARN_API size_t kvarn_decode_workspace_bytes(const kvarn_params* p, int32_t B, int32_t Hq, int32_t Hkv,
                                    int32_t max_chunks);

/*
 * kvarn_quantize_chunk -- the write path for a batch of tiles in ONE launch
 * (Fig. 2: rotate -> VarN -> RTN -> store codes + scale + zero + second
 * scale).  Tile i of K is the 128x128 block at k + i*tile_stride (elements of
 * in_dtype), its token t at + t*tok_stride, channels contiguous; likewise V.
 * Record i is written at k_rec + i*rec_stride (bytes) / v_rec + i*rec_stride.
 *   k, v        DEVICE, in_dtype, 16-B aligned; strides multiples of 8 elements
 *   k_rec,v_rec DEVICE, 16-B aligned; rec_stride >= record_bytes, multiple of 16
 *   dbg         nullable
 * Either of (k, k_rec) or (v, v_rec) may be NULL to quantise only one kind.
 * Precision: fp32 throughout.  Variances are mean-centred; tiles in which a (rotated) channel's mean exceeds
 * four standard deviations take pivoted single-pass sums, so the 1e-5 agreement of the scales with a float64
 * evaluation holds up to channel offsets of ~100 standard deviations; beyond that the fp32 rotation of the input
 * itself (rounding of order |offset| x 2^-24 per butterfly stage) is the limit, not the variance passes.
 * Range: the squares of the values must stay inside fp32 (|x| between ~2^-60 and 2^60); below that the variances
 * underflow to the clamp and the choice of the iterate is no longer the float64 one (the record stays finite).
 */
KVARN_API int kvarn_quantize_chunk(const kvarn_params* p, const void* k, const void* v, int64_t n_tiles,
                         int64_t tile_stride, int64_t tok_stride, void* k_rec, void* v_rec,
                         int64_t rec_stride, const kvarn_debug* dbg, void* stream);

/*
 * kvarn_prefill -- bulk-load a cache from k, v = [B][Hkv][n_tok][128]: copy the
 * first min(n_tok, n_sink) tokens of every (sequence, KV head) into the sink
 * region, quantise the following floor((n_tok - n_sink)/128) chunks into the
 * cache's records, copy the remaining tokens into the residual window and set
 * seq_lens[b] = n_tok.  Same kernel as kvarn_quantize_chunk.
 */
KVARN_API int kvarn_prefill(const kvarn_params* p, const kvarn_cache* cache, const void* k, const void* v,
                  int32_t n_tok, void* stream);

/*
 * kvarn_append -- on-the-fly compression during decoding (P:17, P:53, P:83,
 * P:350): append ONE new token per sequence.  k_new, v_new = [B][Hkv][128]
 * in_dtype (DEVICE).  While len < n_sink the token goes to sink slot len; afterwards
 * (with l = len - n_sink) it goes to residual slot l%128; a residual that
 * thereby reaches 128 tokens is quantised at once into chunk slot l/128 (bit
 * for bit what kvarn_quantize_chunk gives on those 128 tokens) and the residual
 * becomes empty.  seq_lens[b] is read and advanced ON DEVICE (no host round
 * trip).  A sequence already holding n_sink + max_chunks*128 + 127 tokens is left
 * unchanged (its token is dropped): with cache->max_len_hint > 0 the call returns
 * KVARN_CAPACITY instead of launching when the bound proves that a token cannot fit,
 * and a drop the host could not foresee is counted in cache->overflow (if non-null).
 */
KVARN_API int kvarn_append(const kvarn_params* p, const kvarn_cache* cache, const void* k_new,
                 const void* v_new, void* stream);

/*
 * kvarn_append_block -- the same for a block of 1 <= n_new <= 128 tokens per sequence (the write half of a
 * pseudo-decode step, Fig. 4: "After every block, the freshly produced K, V are quantized before being
 * written back to the KV-cache"; kvarn_block_attention is the read half).  k_new, v_new = [B][Hkv][n_new][128]
 * in_dtype (DEVICE).  Tokens fill the sink region first, then the residual window; the (at most one) chunk the
 * window completes is quantised in the same launch, the remaining tokens start the next window.  The result is bit
 * for bit what n_new calls of kvarn_append (or kvarn_prefill of the longer sequence) leave.  A block that does not fit
 * (chunk slot >= max_chunks) leaves the sequence unchanged (KVARN_CAPACITY / cache->overflow as for kvarn_append).
 */
KVARN_API int kvarn_append_block(const kvarn_params* p, const kvarn_cache* cache, const void* k_new,
                       const void* v_new, int32_t n_new, void* stream);

/*
 * kvarn_decode_attention -- out[b][h] = softmax(q[b][h] K^T * sm_scale) V over
 * all seq_lens[b] tokens of KV head h / (Hq/Hkv): the quantised chunks, read as
 * packed codes + scales + zero-points (Eq. 1 with the second scale fused,
 * P:45), the raw sink tokens and the raw residual window.  The Hadamard
 * rotation and the per-channel scales are folded into q and the output.
 *   q    DEVICE [B][Hq][128] in_dtype          out  DEVICE [B][Hq][128] out_dtype
 *   ws   DEVICE scratch of >= kvarn_decode_workspace_bytes(...) bytes, 16-B aligned
 * A sequence of length 0 yields zeros.  Hq/Hkv must be in 1..8.
 * Precision: fp32 accumulation; the folded query and the weights pt = p[t] s1v[t] (probability times the V record's row
 * scale) enter the tensor cores as fixed-point numbers (kvarn_params::decode_digits: 22 / 16 bits by default), the query
 * relative to max_c |q~[h, c]| of its chunk, a weight relative to the largest weight of its own chunk (128 tokens).  A
 * token's VALUE contribution is therefore rounded to zero only if pt lies more than 2^-17 (2^-23 with decode_digits = 4)
 * below the largest of its 127 neighbours -- a bound that does not grow with the context length -- while the
 * denominator takes the exact p, so a token with a tiny V row keeps its probability mass; numerator and denominator
 * differ by at most half a fixed-point unit per token (random sign; worst case 128 x 2^-17 of the chunk's largest
 * weight).  Raw (sink / residual / block) tokens are handled in fp32.
 */
KVARN_API int kvarn_decode_attention(const kvarn_params* p, const kvarn_cache* cache, const void* q,
                           int32_t Hq, float sm_scale, void* out, void* ws, size_t ws_bytes,
                           void* stream);

/*
 * kvarn_decode_attention_static -- kvarn_decode_attention for callers that cannot allocate device memory (code under
 * CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): same operation, arguments, precision and
 * result, but the split-K scratch (arrival counters + workspace partials; cache->decode_ticket is not used and may be
 * NULL) lives in a static device array of KVARN_STATIC_SCRATCH_BYTES (1 MiB) inside the library, which every GPU that
 * loads the library holds until the process exits.  The call allocates nothing (no cudaMalloc / cudaFree / allocating
 * library routine).  Limits: a split plan that needs more than 1 MiB - 4 KiB of partials (B * Hq * clusters-per-sequence
 * * 1040 B; every plan the library chooses itself for <= 8 KV-head groups stays below 0.4 MiB, only caller-chosen
 * kvarn_params::splits can exceed it) or more than 1024 (sequence, KV head) units on the workspace route returns
 * KVARN_WORKSPACE_TOO_SMALL.  ALL calls on one GPU share the array: calls that may overlap on the GPU (different streams
 * without ordering) race; order them on one stream or use kvarn_decode_attention with separate workspaces.  The array
 * keeps the previous call's contents; the call clears the counters it needs on `stream` before the launch.
 * The device of `stream` must be current.  The first call on a device does the one-time set-up (the array's device address,
 * the kernel's shared-memory attribute): make it once before capturing the stream into a graph.
 */
#define KVARN_STATIC_SCRATCH_BYTES (1u << 20)
KVARN_API int kvarn_decode_attention_static(const kvarn_params* p, const kvarn_cache* cache, const void* q,
                                  int32_t Hq, float sm_scale, void* out, void* stream);

/*
 * Context-parallel building block ("Splitting one sequence's chunks across GPUs needs exactly one
 * exchange: all-gather (m, l, acc[128]) per q head and LSE-merge").  Each rank holds a cache over ITS part of every
 * sequence and calls kvarn_decode_attention_partial, which is kvarn_decode_attention stopping before the
 * normalisation: part[b][h] = { m, l, 0, 0, o[128] } (KVARN_PART_STRIDE = 132 fp32), with m a reference exponent
 * in log2 units of the scaled logits (the kernel's running maximum, which includes the folded value scale; -inf for
 * an empty part), l = sum_t 2^(logit_t - m), o = sum_t 2^(logit_t - m) v_t in the caller's (un-rotated) space.  After the ranks all-gather their `part` arrays into parts[n_parts][n_rows][132]
 * (n_rows = B * Hq; one NCCL all-gather), kvarn_merge_partials computes
 *   out[row] = sum_r 2^(m_r - m*) o_r / sum_r 2^(m_r - m*) l_r,   m* = max_r m_r   (zeros if every part is empty).
 * All pointers DEVICE, 16-B aligned; ws as for kvarn_decode_attention.
 */
#define KVARN_PART_STRIDE 132
KVARN_API int kvarn_decode_attention_partial(const kvarn_params* p, const kvarn_cache* cache, const void* q,
                                   int32_t Hq, float sm_scale, float* part, void* ws, size_t ws_bytes,
                                   void* stream);
KVARN_API int kvarn_merge_partials(const float* parts, int32_t n_parts, int64_t n_rows, void* out, int32_t out_dtype,
                         void* stream);

/*
 * kvarn_block_attention -- the multi-token read path (Fig. 4 "pseudo-decode", Sec. 3.2:
 * "We split the sequence into blocks of size b.  After every block, the freshly produced K, V are
 * quantized before being written back to the KV-cache.  Subsequent blocks access a quantized cache").
 * A block of n_q new tokens per sequence (speculative / chunked decoding, 1 <= n_q <= 128) attends
 *   - every token already in the cache (sink tokens, packed chunks, residual window: exactly what
 *     kvarn_decode_attention reads, no dequantised copy), and
 *   - causally, the block's own raw tokens: query i sees block tokens 0..i.
 * The block is NOT in the cache yet; the caller appends it afterwards (kvarn_append per token).
 *   q      DEVICE [B][n_q][Hq][128] in_dtype       out  DEVICE [B][n_q][Hq][128] out_dtype
 *   k_blk, v_blk  DEVICE [B][Hkv][n_q][128] in_dtype (raw, un-rotated), 16-B aligned
 * Hq/Hkv must be 1, 2, 4 or 8.  Needs no workspace (split-K merges inside a thread-block cluster).
 */
KVARN_API int kvarn_block_attention(const kvarn_params* p, const kvarn_cache* cache, const void* q,
                          const void* k_blk, const void* v_blk, int32_t n_q, int32_t Hq,
                          float sm_scale, void* out, void* stream);

/*
 * kvarn_block_attention_dense -- the same operation and arguments as kvarn_block_attention, computed by a dense
 * tensor-core kernel (tcgen05 + tensor memory): every chunk of the cache is expanded once into fp16 tiles
 * (code x scale is exact in fp16) and the block's 128-row tiles of (query token, head) pairs run S = Q K^T and
 * O += P V as M = 128 MMAs; the raw windows (sink, residual, the block's own causal tokens) pass through the same
 * pipeline as fp16 tiles (keys in two fp16 terms, values in one: 2^-12 per element) and the pieces are LSE-merged.  The right
 * form for blocks with >= ~32 (token, head) rows per KV head (blocks of b tokens); kvarn_block_attention is the
 * right one for a few speculative tokens.  ws: DEVICE scratch of >= kvarn_block_dense_workspace_bytes(...) bytes
 * (16-byte aligned; owned by the caller, may be reused by the next call on the same stream).
 * Precision: the query enters as two fp16 terms (22 bits), the tiles are exact (the V row scale s1v[t] enters as its
 * exact mantissa part in the tile and a per-chunk power of two in the logits; a token whose s1v is more than 2^9 below
 * the largest of its chunk loses low bits), probabilities are fp16 relative to 2^8 times the running row maximum, with
 * numerator and denominator from the same rounded values; accumulation in fp32.  Same tolerance as
 * kvarn_block_attention (2e-3 of the output scale).  Errors: as kvarn_block_attention, + KVARN_WORKSPACE_TOO_SMALL.
 */
KVARN_API size_t kvarn_block_dense_workspace_bytes(const kvarn_params* p, int32_t B, int32_t Hq, int32_t Hkv, int32_t n_q,
                                         int32_t max_chunks);
KVARN_API int kvarn_block_attention_dense(const kvarn_params* p, const kvarn_cache* cache, const void* q,
                                const void* k_blk, const void* v_blk, int32_t n_q, int32_t Hq,
                                float sm_scale, void* out, void* ws, size_t ws_bytes, void* stream);

/*
 * The Hadamard arrangement around the attention layer (App. A: "two absorbed transforms (that are
 * merged with W_V and W_O respectively ...) and two online transforms after the RoPE-embedding.  The two online
 * transforms are head-wise").  With these a model can produce q, K and V already rotated and run the cache with
 * rotate_k = rotate_v = 0.  All pointers DEVICE; in place (y == x, out == w) is allowed; dtype = kvarn_dtype.
 *
 * kvarn_rope_hadamard -- the online transform of q or K fused with the rotary embedding:
 *   y[t][h][:] = RoPE(x[t][h][:]) H / sqrt(128),  x, y [n_tok][n_heads][128], 16-B aligned.
 *   cos_tab, sin_tab: fp32 [n_tok][64] of the token's position, half-split convention (channel c < 64 pairs with
 *   c + 64: y[c] = x[c] cos[c] - x[c+64] sin[c], y[c+64] = x[c+64] cos[c] + x[c] sin[c]); both null = no RoPE.
 *   rotate = 0 applies the rotary embedding only.
 * kvarn_hadamard_rows -- every 128-element group of a contiguous array rotated (x [n_groups][128]): the absorbed
 *   transform of W_V stored [d_model][Hkv*128] (W_V' = W_V R), or a plain online rotation.
 * kvarn_hadamard_row_groups -- W' = R^T W for row-major W [n_rows][n_cols], n_rows a multiple of 128: each group
 *   of 128 consecutive rows is rotated down the columns: the absorbed transform of W_O stored [Hq*128][d_model].
 */
KVARN_API int kvarn_rope_hadamard(const void* x, const float* cos_tab, const float* sin_tab, void* y, int64_t n_tok,
                        int32_t n_heads, int32_t dtype, int32_t rotate, void* stream);
KVARN_API int kvarn_hadamard_rows(const void* x, void* y, int64_t n_groups, int32_t dtype, void* stream);
KVARN_API int kvarn_hadamard_row_groups(const void* w, void* out, int64_t n_rows, int64_t n_cols, int32_t dtype,
                              void* stream);

/*
 * Host-buffer forms (end-to-end measurement; HOST pointers in, HOST out).
 * They copy host->device into caller-provided DEVICE staging, run the device
 * call above and copy the result back, all enqueued on `stream`; the caller
 * synchronises the stream before reading the host outputs.
 *   kvarn_quantize_chunk_host: k_host, v_host contiguous [n_tiles][128][128];
 *     dev_in_k / dev_in_v DEVICE staging of the same size; dev_rec_k / dev_rec_v
 *     DEVICE records [n_tiles][record_bytes] (kept: they are the cache);
 *     k_rec_host / v_rec_host nullable HOST copies of the records.
 *   kvarn_decode_attention_host: q_host [B][Hq][128] -> out_host [B][Hq][128];
 *     dev_q / dev_out DEVICE staging.
 */
KVARN_API int kvarn_quantize_chunk_host(const kvarn_params* p, const void* k_host, const void* v_host,
                              int64_t n_tiles, void* dev_in_k, void* dev_in_v, void* dev_rec_k,
                              void* dev_rec_v, void* k_rec_host, void* v_rec_host, void* stream);
KVARN_API int kvarn_decode_attention_host(const kvarn_params* p, const kvarn_cache* cache,
                                const void* q_host, int32_t Hq, float sm_scale, void* out_host,
                                void* dev_q, void* dev_out, void* ws, size_t ws_bytes,
                                void* stream);

/*
 * Test hooks (pure host code, HOST pointers): convert one record to / from the
 * canonical form  codes[t][c] (u8, 128x128, token-major for BOTH kinds),
 * s1[128], s2[128], z[128] as fp32 (exact values of the stored FP8/FP16).
 * s1 and z are indexed by the RTN group (K: channel, V: token), s2 by the
 * other axis.  pack rounds s1/s2 to FP8-E4M3 and z to FP16 (RNE, saturating).
 */
KVARN_API int kvarn_unpack_record_host(const kvarn_params* p, int32_t kind, const void* record,
                             uint8_t* codes, float* s1, float* s2, float* z);
KVARN_API int kvarn_pack_record_host(const kvarn_params* p, int32_t kind, const uint8_t* codes,
                           const float* s1, const float* s2, const float* z, void* record);

#ifdef __cplusplus
}
#endif
#endif /* KVARN_H_ */

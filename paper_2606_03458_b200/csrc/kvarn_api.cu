// C-ABI entry points of libkvarn (include/kvarn.h): argument validation, kernel
// launches on the caller's stream, host-side record pack/unpack test hooks.
#include <atomic>
#include <cstdio>
#include <cstring>

#include "kvarn_common.cuh"
#include "kvarn_decode.cuh"
#include "kvarn_block_dense.cuh"
#include <cstdlib>
#include "kvarn_rotate.cuh"
#include "kvarn_quantize.cuh"

namespace kvarn {

// ------------------------------------------------------------------ kernels
struct QuantArgs {
  const void* in[2];
  uint8_t* rec[2];
  long long n_inner;
  long long in_base;                                       // elements: first tile starts here (after the sink tokens)
  long long in_outer_stride, in_tile_stride, tok_stride;  // elements
  long long rec_outer_stride, rec_stride;                 // bytes
  long long n_tiles;
  int kind_base;
  int rotate[2];
  VarnConsts vc;
  int32_t* dbg_kbest;
  float* dbg_imb;
  float* dbg_aux;
};

template <int BITS, typename InT>
__global__ void __launch_bounds__(256, 2) quantize_kernel(const QuantArgs A) {
  extern __shared__ __align__(16) uint8_t quant_smem_raw[];
  QuantSmem<BITS>& sm = *reinterpret_cast<QuantSmem<BITS>*>(quant_smem_raw);
  const int kind = A.kind_base + blockIdx.y;
  const long long tile = blockIdx.x;
  const long long outer = tile / A.n_inner, inner = tile - outer * A.n_inner;
  const InT* src = reinterpret_cast<const InT*>(A.in[kind]) + A.in_base + outer * A.in_outer_stride +
                   inner * A.in_tile_stride;
  uint8_t* dst = A.rec[kind] + outer * A.rec_outer_stride + inner * A.rec_stride;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int c0 = 8 * (lane & 15), t0 = 16 * warp + 8 * (lane >> 4);
  float2 x[8][4];
#pragma unroll
  for (int i = 0; i < 8; ++i) load_row8<InT>(src + (long long)(t0 + i) * A.tok_stride + c0, x[i]);
  QuantDebug dbg;
  dbg.k_best = A.dbg_kbest ? A.dbg_kbest + (long long)kind * A.n_tiles : nullptr;
  dbg.imb = A.dbg_imb ? A.dbg_imb + (long long)kind * A.n_tiles * (KVARN_MAX_ITERS + 1) : nullptr;
  dbg.aux = A.dbg_aux ? A.dbg_aux + (long long)kind * A.n_tiles * 384 : nullptr;
  quantize_tile<BITS>(x, kind, A.rotate[kind] != 0, A.vc, dst, dbg, tile, sm);
}

struct AppendArgs {
  uint8_t* rec[2];
  void* resid[2];
  const void* tok[2];
  void* sink[2];
  int32_t* seq_lens;
  int32_t* ticket;
  int32_t* overflow;   // nullable: sticky count of (sequence, call) pairs whose tokens were dropped
  int B, Hkv, max_chunks, n_sink;
  int n_new;   // tokens appended per sequence (1..128); tok = [B][Hkv][n_new][128]
  int rotate[2];
  VarnConsts vc;
};

// One CTA per (sequence, KV head, kind) appends n_new <= 128 tokens (kvarn_append: 1).  The decision to quantise
// is taken on the device from seq_lens (no host round trip).  Three-region layout of P:350: tokens go to
// the sink while len < n_sink, then to the residual window; since the window holds < 128 tokens and n_new <= 128 at
// most one chunk completes: it is quantised from [window rows ; new tokens] and the rest starts the next window.
template <int BITS, typename InT>
__global__ void __launch_bounds__(256, 2) append_kernel(const AppendArgs A) {
  extern __shared__ __align__(16) uint8_t quant_smem_raw[];
  QuantSmem<BITS>& sm = *reinterpret_cast<QuantSmem<BITS>*>(quant_smem_raw);
  const int kind = blockIdx.y, bh = blockIdx.x, b = bh / A.Hkv;
  const int tid = threadIdx.x;
  const int n = A.n_new;
  const int len = A.seq_lens[b];
  const int n_s = min(max(A.n_sink - len, 0), n);     // new tokens that still belong to the sink region
  const int nb = n - n_s;                             // new tokens of the body
  const int l0 = max(len - A.n_sink, 0);              // body tokens already stored
  const int r0 = l0 & 127, chunk = l0 >> 7;
  const bool full = nb > 0 && r0 + nb >= G;           // the window completes a chunk
  const bool can_store = nb == 0 || (full ? (chunk < A.max_chunks) : (chunk <= A.max_chunks));
  InT* resid = reinterpret_cast<InT*>(A.resid[kind]) + (size_t)bh * G * D;
  const InT* tok = reinterpret_cast<const InT*>(A.tok[kind]) + (size_t)bh * n * D;
  if (can_store) {
    if (n_s > 0) {
      InT* sink = reinterpret_cast<InT*>(A.sink[kind]) + ((size_t)bh * A.n_sink + len) * D;
      for (int i = tid; i < n_s * D; i += 256) sink[i] = tok[i];
    }
    const InT* btok = tok + (size_t)n_s * D;          // first body token of the block
    if (!full) {
      for (int i = tid; i < nb * D; i += 256) resid[(size_t)r0 * D + i] = btok[i];
    } else {
      const int lane = tid & 31, warp = tid >> 5;
      const int c0 = 8 * (lane & 15), t0 = 16 * warp + 8 * (lane >> 4);
      float2 x[8][4];
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int t = t0 + i;
        const InT* row = (t < r0) ? resid + (size_t)t * D : btok + (size_t)(t - r0) * D;
        load_row8<InT>(row + c0, x[i]);
      }
      uint8_t* dst = A.rec[kind] + ((size_t)bh * A.max_chunks + chunk) * record_bytes(BITS);
      QuantDebug dbg{nullptr, nullptr, nullptr};
      quantize_tile<BITS>(x, kind, A.rotate[kind] != 0, A.vc, dst, dbg, 0, sm);   // (barriers inside: every row is loaded)
      const int rem = r0 + nb - G;                    // tokens that start the next window
      const InT* rtok = btok + (size_t)(G - r0) * D;
      for (int i = tid; i < rem * D; i += 256) resid[i] = rtok[i];
    }
  }
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    const int old = atomicAdd(&A.ticket[b], 1);
    if (old == 2 * A.Hkv - 1) {  // last CTA of this sequence: every CTA has read seq_lens[b]
      A.ticket[b] = 0;
      if (can_store) A.seq_lens[b] = len + n;
      else if (A.overflow) atomicAdd(A.overflow, 1);
    }
  }
}

struct TailArgs {
  const void* in[2];
  void* resid[2];
  void* sink[2];
  int32_t* seq_lens;
  int B, Hkv, n_tok, n_full, n_sink;
};
// raw regions of a bulk load: the first min(n_tok, n_sink) tokens -> sink, the tokens after the full chunks -> residual
template <typename InT>
__global__ void prefill_tail_kernel(const TailArgs A) {
  const int bh = blockIdx.x, kind = blockIdx.y;
  const int ns = min(A.n_tok, A.n_sink);
  const int r = A.n_tok - ns - A.n_full * G;
  const InT* base = reinterpret_cast<const InT*>(A.in[kind]) + (size_t)bh * A.n_tok * D;
  if (ns > 0) {
    InT* sdst = reinterpret_cast<InT*>(A.sink[kind]) + (size_t)bh * A.n_sink * D;
    for (int i = threadIdx.x; i < ns * D; i += blockDim.x) sdst[i] = base[i];
  }
  const InT* src = base + ((size_t)ns + (size_t)A.n_full * G) * D;
  InT* dst = reinterpret_cast<InT*>(A.resid[kind]) + (size_t)bh * G * D;
  for (int i = threadIdx.x; i < r * D; i += blockDim.x) dst[i] = src[i];
  if (kind == 0 && threadIdx.x == 0 && (bh % A.Hkv) == 0) A.seq_lens[bh / A.Hkv] = A.n_tok;
}

// ------------------------------------------------------------------ host helpers
static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

static int check_params(const kvarn_params* p) {
  if (!p) return KVARN_INVALID_ARG;
  if (p->head_dim != D || p->chunk != G) return KVARN_UNSUPPORTED;
  if (p->bits != 2 && p->bits != 4) return KVARN_UNSUPPORTED;
  if (p->iters < 0 || p->iters > KVARN_MAX_ITERS) return KVARN_INVALID_ARG;
  if (p->aux_round != 0 && p->aux_round != 1) return KVARN_INVALID_ARG;
  if (p->decode_digits != 0 && p->decode_digits != 2 && p->decode_digits != 4) return KVARN_INVALID_ARG;
  if (p->in_dtype != KVARN_BF16 && p->in_dtype != KVARN_F32) return KVARN_UNSUPPORTED;
  if (p->out_dtype != KVARN_BF16 && p->out_dtype != KVARN_F32) return KVARN_UNSUPPORTED;
  if (!(p->var_min > 0.f) || !(p->var_max >= p->var_min) || !(p->log_hi >= p->log_lo)) return KVARN_INVALID_ARG;
  return KVARN_OK;
}

static VarnConsts varn_consts(const kvarn_params* p) {
  VarnConsts vc;
  vc.iters = p->iters; vc.var_min = p->var_min; vc.var_max = p->var_max;
  vc.log_lo = p->log_lo; vc.log_hi = p->log_hi;
  vc.aux_round = p->aux_round;
  return vc;
}

static int last_cuda() { return cudaGetLastError() == cudaSuccess ? KVARN_OK : KVARN_CUDA; }

// The device the launch goes to: CUDA launches on the CURRENT device (the caller's stream must belong to it).
static int current_device() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return -1; }
  return dev;
}

// Opt-in to more than 48 KB of dynamic shared memory (+ the shared-memory carve-out).  The attribute belongs to
// the (kernel, device) pair, so it is applied once PER DEVICE: a bit mask indexed by the current device, one mask
// per kernel (KERN is a template argument).  Atomic: two host threads may race here, the call is idempotent.
constexpr int KVARN_MAX_DEVICES = 64;
template <auto KERN>
static cudaError_t ensure_smem_optin(int bytes, bool max_carveout) {
  static std::atomic<uint64_t> done{0};
  const int dev = current_device();
  if (dev < 0) return cudaErrorNoDevice;
  if (dev < KVARN_MAX_DEVICES && ((done.load(std::memory_order_acquire) >> dev) & 1)) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(KERN, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e != cudaSuccess) return e;
  if (max_carveout) {
    e = cudaFuncSetAttribute(KERN, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
  }
  if (dev < KVARN_MAX_DEVICES) done.fetch_or(1ull << dev, std::memory_order_release);
  return cudaSuccess;
}

// QuantSmem exceeds the 48 KB static limit: dynamic, opt-in
template <int BITS, auto KERN, typename Args>
static int launch_quant_smem(dim3 grid, const Args& A, cudaStream_t st) {
  if (ensure_smem_optin<KERN>((int)sizeof(QuantSmem<BITS>), false) != cudaSuccess) { cudaGetLastError(); return KVARN_CUDA; }
  KERN<<<grid, dim3(256), sizeof(QuantSmem<BITS>), st>>>(A);
  return last_cuda();
}

static int launch_quantize(const kvarn_params* p, const QuantArgs& A, int n_kinds, cudaStream_t st) {
  if (A.n_tiles == 0) return KVARN_OK;
  dim3 grid((unsigned)A.n_tiles, (unsigned)n_kinds);
  const bool f32 = p->in_dtype == KVARN_F32;
  if (p->bits == 2) {
    if (f32) return launch_quant_smem<2, quantize_kernel<2, float>>(grid, A, st);
    return launch_quant_smem<2, quantize_kernel<2, __nv_bfloat16>>(grid, A, st);
  }
  if (f32) return launch_quant_smem<4, quantize_kernel<4, float>>(grid, A, st);
  return launch_quant_smem<4, quantize_kernel<4, __nv_bfloat16>>(grid, A, st);
}

// Split-K plan of kvarn_decode_attention: `cluster` CTAs of a thread-block cluster share one
// (sequence, KV head) and merge through DSMEM; `nclus` clusters per (sequence, KV head) merge
// through the workspace (only when one cluster leaves most of the GPU idle on long contexts).
struct SplitPlan { int cluster, nclus; };
#ifndef KVARN_SPLIT_FEW_SLOTS
#define KVARN_SPLIT_FEW_SLOTS 2
#endif
#ifndef KVARN_MAX_CLUSTER_OVERRIDE
#define KVARN_MAX_CLUSTER_OVERRIDE 8
#endif
constexpr int KVARN_DENSE_CTA_COST = 14;    // fixed cost of a dense CTA / of the merge launch, in chunk-times (~2 us each)
constexpr int KVARN_DENSE_MERGE_COST = 12;
constexpr int KVARN_MAX_CLUSTER = KVARN_MAX_CLUSTER_OVERRIDE;    // portable maximum; 9..16 (non-portable) measured slower: 25 -> 27..31 us on config 1

// DQ, DP = digit planes of q~ / p~ (kvarn_decode.cuh)
template <int BITS, int GP, int DQ, int DP, typename InT>
struct DecKernel {
  static constexpr size_t smem = sizeof(DecSmemW<BITS, GP, DQ, DP>);
  static auto kern() { return decode_kernel_w<BITS, GP, DQ, DP, InT>; }
  static cudaError_t optin() { return ensure_smem_optin<decode_kernel_w<BITS, GP, DQ, DP, InT>>((int)smem, true); }
};

// Calls f(DecKernel<...>{}) for the instantiation that serves (params, gp = 4 | 8 columns per CTA).
// kvarn_params::decode_digits: 0 = (DQ, DP) = (4, 2), 2 = (2, 2) [4-bit caches: (4, 2)], 4 = (4, 4).
template <class F>
static auto with_decode_kernel(const kvarn_params* p, int gp, F&& f) {
  const bool f32 = p->in_dtype == KVARN_F32;
  const int dig = p->decode_digits;
  if (p->bits == 2) {
    if (gp == 4) {
      if (dig == 2) return f32 ? f(DecKernel<2, 4, 2, 2, float>{}) : f(DecKernel<2, 4, 2, 2, __nv_bfloat16>{});
      if (dig == 4) return f32 ? f(DecKernel<2, 4, 4, 4, float>{}) : f(DecKernel<2, 4, 4, 4, __nv_bfloat16>{});
      return f32 ? f(DecKernel<2, 4, 4, 2, float>{}) : f(DecKernel<2, 4, 4, 2, __nv_bfloat16>{});
    }
    if (dig == 2) return f32 ? f(DecKernel<2, 8, 2, 2, float>{}) : f(DecKernel<2, 8, 2, 2, __nv_bfloat16>{});
    if (dig == 4) return f32 ? f(DecKernel<2, 8, 4, 4, float>{}) : f(DecKernel<2, 8, 4, 4, __nv_bfloat16>{});
    return f32 ? f(DecKernel<2, 8, 4, 2, float>{}) : f(DecKernel<2, 8, 4, 2, __nv_bfloat16>{});
  }
  if (gp == 4) {
    if (dig == 4) return f32 ? f(DecKernel<4, 4, 4, 4, float>{}) : f(DecKernel<4, 4, 4, 4, __nv_bfloat16>{});
    return f32 ? f(DecKernel<4, 4, 4, 2, float>{}) : f(DecKernel<4, 4, 4, 2, __nv_bfloat16>{});
  }
  if (dig == 4) return f32 ? f(DecKernel<4, 8, 4, 4, float>{}) : f(DecKernel<4, 8, 4, 4, __nv_bfloat16>{});
  return f32 ? f(DecKernel<4, 8, 4, 2, float>{}) : f(DecKernel<4, 8, 4, 2, __nv_bfloat16>{});
}

// resident CTAs of the decode kernel per SM on the current device (cached per device and instantiation)
template <class DK>
static int decode_ctas_per_sm(DK) {
  static std::atomic<int> cached[KVARN_MAX_DEVICES] = {};
  const int dev = current_device();
  const int fallback = 3;   // no device (host-only queries): a conservative constant
  if (dev < 0) return fallback;
  if (dev < KVARN_MAX_DEVICES) { const int c = cached[dev].load(std::memory_order_relaxed); if (c) return c; }
  int n = 0;
  if (DK::optin() != cudaSuccess ||
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, DK::kern(), 128, DK::smem) != cudaSuccess || n < 1) {
    cudaGetLastError();
    return fallback;
  }
  if (dev < KVARN_MAX_DEVICES) cached[dev].store(n, std::memory_order_relaxed);
  return n;
}
static int decode_slots(const kvarn_params* p, int g) {
  int sms = 148;
  const int dev = current_device();   // = the device of the caller's stream (CUDA requires it to be current)
  if (dev >= 0 && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) { cudaGetLastError(); sms = 148; }
  return sms * with_decode_kernel(p, g <= 4 ? 4 : 8, [](auto dk) { return decode_ctas_per_sm(dk); });
}

static SplitPlan split_plan(const kvarn_params* p, int B, int Hkv, int g, int max_chunks) {
  SplitPlan sp{1, 1};
  if (max_chunks <= 1) return sp;
  if (p->splits > 0) {   // caller-chosen total: the largest cluster size (<= 8) that divides it
    int s = p->splits < max_chunks ? p->splits : max_chunks;
    int cs = KVARN_MAX_CLUSTER;
    while (s % cs) --cs;
    sp.cluster = cs; sp.nclus = s / cs;
    if (sp.nclus > 64) sp.nclus = 64;
    return sp;
  }
  const int bh = B * Hkv;
  const int slots = decode_slots(p, g);        // resident CTAs of the decode kernel on this device
  int want = slots / bh;                        // splits that still fit in one wave
  if (want < 1) want = 1;
  if (want > max_chunks) want = max_chunks;
  sp.cluster = want < KVARN_MAX_CLUSTER ? want : KVARN_MAX_CLUSTER;
  // at least one chunk per warp of every CTA: below that the cluster's launch and merge cost more than they spread
  // (B = 8, 8 KV heads, 1024 tokens: 11.2 us with 8 CTAs per unit, 8.6 with 2)
  if (sp.cluster > 1 && max_chunks < 4 * sp.cluster) sp.cluster = max_chunks >= 8 ? max_chunks / 4 : 1;
  // about one CTA per slot and long CTAs: halve them, so that the CTAs of the second half-wave balance the SMs that
  // got one CTA more (config 4, 512 units on 444 slots: 1 / 2 / 3 / 4 / 6 CTAs per unit measured in DESIGN.md 6.2)
  if (sp.cluster == 1 && max_chunks >= 32) sp.cluster = KVARN_SPLIT_FEW_SLOTS;
  if (sp.cluster == KVARN_MAX_CLUSTER) {
    const int per = (max_chunks + KVARN_MAX_CLUSTER - 1) / KVARN_MAX_CLUSTER;   // chunks per CTA with one cluster
    if (per > 32) {   // a very long context with few sequences: several clusters per sequence, merged through the workspace
      int nc = want / KVARN_MAX_CLUSTER, cap = per / 16;
      if (nc > cap) nc = cap;
      if (nc > 64) nc = 64;
      if (nc > 1) sp.nclus = nc;
    }
  }
  return sp;
}

template <class DK>
static cudaError_t launch_decode_k(DK, const DecodeArgs& A, cudaStream_t st) {
  auto kern = DK::kern();
  {
    const cudaError_t e = DK::optin();
    if (e != cudaSuccess) return e;
  }
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(A.B * A.Hkv, A.splits, (A.n_q + A.tpc - 1) / A.tpc);
  cfg.blockDim = dim3(128, 1, 1);
  cfg.dynamicSmemBytes = DK::smem;
  cfg.stream = st;
  // attr[0]: programmatic dependent launch (the kernel waits with griddepcontrol.wait before its first global access:
  // launch latency and CTA scheduling overlap the tail of the previous kernel of the stream); attr[1]: the cluster
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  attr[1].id = cudaLaunchAttributeClusterDimension;
  attr[1].val.clusterDim.x = 1; attr[1].val.clusterDim.y = (unsigned)A.cluster; attr[1].val.clusterDim.z = 1;
  cfg.attrs = attr; cfg.numAttrs = A.cluster > 1 ? 2 : 1;
  return cudaLaunchKernelEx(&cfg, kern, A);
}

static cudaError_t launch_decode(const kvarn_params* p, DecodeArgs& A, cudaStream_t st) {
  A.shl_mul[0] = 4u; A.shl_mul[1] = 16u; A.shl_mul[2] = 64u;
  return with_decode_kernel(p, A.tpc * A.g <= 4 ? 4 : 8, [&](auto dk) { return launch_decode_k(dk, A, st); });
}

}  // namespace kvarn

using namespace kvarn;

// ------------------------------------------------------------------ C ABI
extern "C" {

void kvarn_default_params(kvarn_params* p, int32_t bits) {
  if (!p) return;
  memset(p, 0, sizeof(*p));
  p->head_dim = D; p->chunk = G; p->bits = bits; p->iters = 8;
  p->var_min = 1e-8f; p->var_max = 1e8f; p->log_lo = -0.3f; p->log_hi = 10.0f;
  p->rotate_k = 1; p->rotate_v = 1;
  p->in_dtype = KVARN_BF16; p->out_dtype = KVARN_F32; p->splits = 0;
}

const char* kvarn_status_string(int status) {
  switch (status) {
    case KVARN_OK: return "KVARN_OK";
    case KVARN_INVALID_ARG: return "KVARN_INVALID_ARG";
    case KVARN_UNSUPPORTED: return "KVARN_UNSUPPORTED";
    case KVARN_MISALIGNED: return "KVARN_MISALIGNED";
    case KVARN_WORKSPACE_TOO_SMALL: return "KVARN_WORKSPACE_TOO_SMALL";
    case KVARN_CAPACITY: return "KVARN_CAPACITY";
    case KVARN_CUDA: return "KVARN_CUDA";
    default: return "KVARN_UNKNOWN_STATUS";
  }
}

int kvarn_version(void) { return 3; }

int kvarn_layout(const kvarn_params* p, kvarn_layout_info* out) {
  if (!p || !out) return KVARN_INVALID_ARG;
  if (p->bits != 2 && p->bits != 4) return KVARN_UNSUPPORTED;
  out->record_bytes = record_bytes(p->bits);
  out->codes_off = 0; out->codes_bytes = codes_bytes(p->bits);
  out->s1_off = s1_off(p->bits); out->s2_off = s2_off(p->bits); out->z_off = z_off(p->bits);
  return KVARN_OK;
}

size_t kvarn_decode_workspace_bytes(const kvarn_params* p, int32_t B, int32_t Hq, int32_t Hkv,
                                    int32_t max_chunks) {
  if (!p || B <= 0 || Hq <= 0 || Hkv <= 0) return 0;
  const SplitPlan sp = split_plan(p, B, Hkv, Hq / Hkv, max_chunks);
  return (size_t)B * Hq * sp.nclus * WS_STRIDE * sizeof(float);   // read and written only when nclus > 1
}

int kvarn_quantize_chunk(const kvarn_params* p, const void* k, const void* v, int64_t n_tiles,
                         int64_t tile_stride, int64_t tok_stride, void* k_rec, void* v_rec,
                         int64_t rec_stride, const kvarn_debug* dbg, void* stream) {
  int st = check_params(p);
  if (st) return st;
  if (n_tiles == 0) return KVARN_OK;
  const bool do_k = k && k_rec, do_v = v && v_rec;
  if (n_tiles < 0 || (!do_k && !do_v) || (k && !k_rec) || (v && !v_rec) || (!k && k_rec) || (!v && v_rec))
    return KVARN_INVALID_ARG;
  if (n_tiles > 0x7fffffffLL) return KVARN_CAPACITY;
  if (tok_stride < D || tile_stride < 0) return KVARN_INVALID_ARG;
  if ((tok_stride % 8) || (tile_stride % 8) || (rec_stride % 16) || !aligned16(k) || !aligned16(v) ||
      !aligned16(k_rec) || !aligned16(v_rec))
    return KVARN_MISALIGNED;
  if (rec_stride < (int64_t)record_bytes(p->bits)) return KVARN_INVALID_ARG;
  QuantArgs A{};
  A.in[0] = k; A.in[1] = v; A.rec[0] = (uint8_t*)k_rec; A.rec[1] = (uint8_t*)v_rec;
  A.n_inner = n_tiles > 0 ? n_tiles : 1; A.in_outer_stride = 0; A.in_tile_stride = tile_stride;
  A.tok_stride = tok_stride; A.rec_outer_stride = 0; A.rec_stride = rec_stride; A.n_tiles = n_tiles;
  A.kind_base = do_k ? 0 : 1;
  A.rotate[0] = p->rotate_k; A.rotate[1] = p->rotate_v;
  A.vc = varn_consts(p);
  if (dbg) { A.dbg_kbest = dbg->k_best; A.dbg_imb = dbg->imb; A.dbg_aux = dbg->aux_f32; }
  return launch_quantize(p, A, (do_k && do_v) ? 2 : 1, (cudaStream_t)stream);
}

static int check_cache(const kvarn_cache* c) {
  if (!c || !c->k_records || !c->v_records || !c->k_resid || !c->v_resid || !c->seq_lens) return KVARN_INVALID_ARG;
  if (c->B <= 0 || c->Hkv <= 0 || c->max_chunks < 0) return KVARN_INVALID_ARG;
  if (c->n_sink < 0 || c->n_sink > G) return KVARN_UNSUPPORTED;
  if (c->n_sink > 0 && (!c->k_sink || !c->v_sink)) return KVARN_INVALID_ARG;
  if (c->n_sink > 0 && (!aligned16(c->k_sink) || !aligned16(c->v_sink))) return KVARN_MISALIGNED;
  if (!aligned16(c->k_records) || !aligned16(c->v_records) || !aligned16(c->k_resid) || !aligned16(c->v_resid))
    return KVARN_MISALIGNED;
  return KVARN_OK;
}

int kvarn_prefill(const kvarn_params* p, const kvarn_cache* cache, const void* k, const void* v,
                  int32_t n_tok, void* stream) {
  int st = check_params(p);
  if (st) return st;
  if ((st = check_cache(cache))) return st;
  if (n_tok < 0 || ((!k || !v) && n_tok > 0)) return KVARN_INVALID_ARG;
  if (!aligned16(k) || !aligned16(v)) return KVARN_MISALIGNED;
  const int ns = n_tok < cache->n_sink ? n_tok : cache->n_sink;
  const int n_full = (n_tok - ns) / G;
  if (n_full > cache->max_chunks) return KVARN_CAPACITY;
  const long long BH = (long long)cache->B * cache->Hkv;
  if (BH * n_full > 0x7fffffffLL) return KVARN_CAPACITY;
  cudaStream_t s = (cudaStream_t)stream;
  QuantArgs A{};
  A.in[0] = k; A.in[1] = v; A.rec[0] = (uint8_t*)cache->k_records; A.rec[1] = (uint8_t*)cache->v_records;
  A.n_inner = n_full > 0 ? n_full : 1;
  A.in_base = (long long)ns * D;
  A.in_outer_stride = (long long)n_tok * D; A.in_tile_stride = (long long)G * D; A.tok_stride = D;
  A.rec_outer_stride = (long long)cache->max_chunks * record_bytes(p->bits);
  A.rec_stride = record_bytes(p->bits);
  A.n_tiles = BH * n_full; A.kind_base = 0;
  A.rotate[0] = p->rotate_k; A.rotate[1] = p->rotate_v; A.vc = varn_consts(p);
  if ((st = launch_quantize(p, A, 2, s))) return st;
  TailArgs T{};
  T.in[0] = k; T.in[1] = v; T.resid[0] = cache->k_resid; T.resid[1] = cache->v_resid;
  T.sink[0] = cache->k_sink; T.sink[1] = cache->v_sink; T.n_sink = cache->n_sink;
  T.seq_lens = cache->seq_lens; T.B = cache->B; T.Hkv = cache->Hkv; T.n_tok = n_tok; T.n_full = n_full;
  dim3 grid((unsigned)BH, 2);
  if (p->in_dtype == KVARN_F32) prefill_tail_kernel<float><<<grid, 256, 0, s>>>(T);
  else prefill_tail_kernel<__nv_bfloat16><<<grid, 256, 0, s>>>(T);
  return last_cuda();
}

int kvarn_append(const kvarn_params* p, const kvarn_cache* cache, const void* k_new,
                 const void* v_new, void* stream) {
  return kvarn_append_block(p, cache, k_new, v_new, 1, stream);
}

int kvarn_append_block(const kvarn_params* p, const kvarn_cache* cache, const void* k_new,
                       const void* v_new, int32_t n_new, void* stream) {
  int st = check_params(p);
  if (st) return st;
  if ((st = check_cache(cache))) return st;
  if (!k_new || !v_new || !cache->ticket || n_new < 1) return KVARN_INVALID_ARG;
  if (n_new > G) return KVARN_UNSUPPORTED;
  if (!aligned16(k_new) || !aligned16(v_new)) return KVARN_MISALIGNED;
  // host-checkable capacity bound: a sequence holds at most n_sink + max_chunks * 128 + 127 tokens
  if (cache->max_len_hint > 0 &&
      (long long)cache->max_len_hint + n_new > (long long)cache->n_sink + (long long)cache->max_chunks * G + (G - 1))
    return KVARN_CAPACITY;
  AppendArgs A{};
  A.rec[0] = (uint8_t*)cache->k_records; A.rec[1] = (uint8_t*)cache->v_records;
  A.resid[0] = cache->k_resid; A.resid[1] = cache->v_resid;
  A.tok[0] = k_new; A.tok[1] = v_new;
  A.seq_lens = cache->seq_lens; A.ticket = cache->ticket; A.overflow = cache->overflow;
  A.sink[0] = cache->k_sink; A.sink[1] = cache->v_sink; A.n_sink = cache->n_sink;
  A.B = cache->B; A.Hkv = cache->Hkv; A.max_chunks = cache->max_chunks; A.n_new = n_new;
  A.rotate[0] = p->rotate_k; A.rotate[1] = p->rotate_v; A.vc = varn_consts(p);
  dim3 grid((unsigned)(cache->B * cache->Hkv), 2);
  cudaStream_t s = (cudaStream_t)stream;
  const bool f32 = p->in_dtype == KVARN_F32;
  if (p->bits == 2) {
    if (f32) return launch_quant_smem<2, append_kernel<2, float>>(grid, A, s);
    return launch_quant_smem<2, append_kernel<2, __nv_bfloat16>>(grid, A, s);
  }
  if (f32) return launch_quant_smem<4, append_kernel<4, float>>(grid, A, s);
  return launch_quant_smem<4, append_kernel<4, __nv_bfloat16>>(grid, A, s);
}

static int decode_impl(const kvarn_params* p, const kvarn_cache* cache, const void* q, int32_t Hq, float sm_scale,
                       void* out, void* ws, size_t ws_bytes, void* stream, int partial) {
  int st = check_params(p);
  if (st) return st;
  if ((st = check_cache(cache))) return st;
  if (!q || !out || !ws || !cache->decode_ticket || Hq <= 0 || (Hq % cache->Hkv) != 0) return KVARN_INVALID_ARG;
  const int g = Hq / cache->Hkv;
  if (g > 8) return KVARN_UNSUPPORTED;
  if (!aligned16(q) || !aligned16(out) || !aligned16(ws)) return KVARN_MISALIGNED;
  const size_t need = kvarn_decode_workspace_bytes(p, cache->B, Hq, cache->Hkv, cache->max_chunks);
  if (ws_bytes < need) return KVARN_WORKSPACE_TOO_SMALL;
  DecodeArgs A{};
  A.k_records = (const uint8_t*)cache->k_records; A.v_records = (const uint8_t*)cache->v_records;
  A.k_resid = cache->k_resid; A.v_resid = cache->v_resid; A.seq_lens = cache->seq_lens;
  A.k_sink = cache->k_sink; A.v_sink = cache->v_sink; A.n_sink = cache->n_sink;
  A.ticket = cache->decode_ticket;
  A.q = q; A.out = out; A.ws = (float*)ws;
  A.B = cache->B; A.Hkv = cache->Hkv; A.Hq = Hq; A.g = g; A.max_chunks = cache->max_chunks;
  const SplitPlan sp = split_plan(p, cache->B, cache->Hkv, g, cache->max_chunks);
  A.cluster = sp.cluster; A.nclus = sp.nclus; A.splits = sp.cluster * sp.nclus;
  A.q_scale = sm_scale * 1.4426950408889634f;
  A.rotate_k = p->rotate_k; A.rotate_v = p->rotate_v; A.out_dtype = p->out_dtype;
  A.n_q = 1; A.tpc = 1; A.k_blk = nullptr; A.v_blk = nullptr; A.partial = partial;
  const cudaError_t e = launch_decode(p, A, (cudaStream_t)stream);
  return e == cudaSuccess ? KVARN_OK : KVARN_CUDA;
}

int kvarn_decode_attention(const kvarn_params* p, const kvarn_cache* cache, const void* q,
                           int32_t Hq, float sm_scale, void* out, void* ws, size_t ws_bytes,
                           void* stream) {
  return decode_impl(p, cache, q, Hq, sm_scale, out, ws, ws_bytes, stream, 0);
}

int kvarn_decode_attention_partial(const kvarn_params* p, const kvarn_cache* cache, const void* q,
                                   int32_t Hq, float sm_scale, float* part, void* ws, size_t ws_bytes,
                                   void* stream) {
  return decode_impl(p, cache, q, Hq, sm_scale, part, ws, ws_bytes, stream, 1);
}

// ---- kvarn_decode_attention_static: the read path for callers that cannot allocate -------------------------------
// The split-K scratch of the decode kernel (arrival counters + workspace partials, touched only when a sequence's
// chunks are spread over several clusters) lives in ONE file-scope device array of KVARN_STATIC_SCRATCH_BYTES per GPU,
// held from the moment the library is loaded on that GPU until the process exits.  In host code the array's NAME is a
// host-side stand-in, not a device address: its device address is taken once per device with cudaGetSymbolAddress
// (that device current) and passed to the kernel.  Layout: [0, 4096) bytes = 1024 int32 arrival counters,
// [4096, KVARN_STATIC_SCRATCH_BYTES) = partials.
static __device__ __align__(256) unsigned char g_static_scratch[KVARN_STATIC_SCRATCH_BYTES];
constexpr size_t STATIC_TICKET_BYTES = 4096;

static cudaError_t static_scratch_ptr(unsigned char** out) {
  static std::atomic<unsigned char*> cached[KVARN_MAX_DEVICES] = {};
  const int dev = current_device();
  if (dev < 0) return cudaErrorInvalidDevice;
  if (dev < KVARN_MAX_DEVICES) { unsigned char* c = cached[dev].load(std::memory_order_acquire); if (c) { *out = c; return cudaSuccess; } }
  unsigned char* ptr = nullptr;
  const cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_static_scratch);   // the current device's copy of the array
  if (e != cudaSuccess || !ptr) { cudaGetLastError(); return e != cudaSuccess ? e : cudaErrorInvalidSymbol; }
  if (dev < KVARN_MAX_DEVICES) cached[dev].store(ptr, std::memory_order_release);
  *out = ptr;
  return cudaSuccess;
}

int kvarn_decode_attention_static(const kvarn_params* p, const kvarn_cache* cache, const void* q,
                                  int32_t Hq, float sm_scale, void* out, void* stream) {
  int st = check_params(p);
  if (st) return st;
  if ((st = check_cache(cache))) return st;
  if (!q || !out || Hq <= 0 || (Hq % cache->Hkv) != 0) return KVARN_INVALID_ARG;
  const int g = Hq / cache->Hkv;
  if (g > 8) return KVARN_UNSUPPORTED;
  if (!aligned16(q) || !aligned16(out)) return KVARN_MISALIGNED;
  const SplitPlan sp = split_plan(p, cache->B, cache->Hkv, g, cache->max_chunks);
  const size_t need = sp.nclus > 1 ? (size_t)cache->B * Hq * sp.nclus * WS_STRIDE * sizeof(float) : 0;
  if (need > KVARN_STATIC_SCRATCH_BYTES - STATIC_TICKET_BYTES ||
      (sp.nclus > 1 && (size_t)cache->B * cache->Hkv * sizeof(int32_t) > STATIC_TICKET_BYTES))
    return KVARN_WORKSPACE_TOO_SMALL;       // the plan needs more scratch than the static array holds
  unsigned char* scratch = nullptr;
  if (static_scratch_ptr(&scratch) != cudaSuccess) return KVARN_CUDA;
  cudaStream_t s = (cudaStream_t)stream;
  // The array keeps the last call's contents.  The partials are written before they are read; the arrival counters must
  // start at zero (a kernel leaves them zero, an aborted or overlapping call may not have): cleared on the stream.
  if (sp.nclus > 1 && cudaMemsetAsync(scratch, 0, (size_t)cache->B * cache->Hkv * sizeof(int32_t), s) != cudaSuccess) {
    cudaGetLastError();
    return KVARN_CUDA;
  }
  DecodeArgs A{};
  A.k_records = (const uint8_t*)cache->k_records; A.v_records = (const uint8_t*)cache->v_records;
  A.k_resid = cache->k_resid; A.v_resid = cache->v_resid; A.seq_lens = cache->seq_lens;
  A.k_sink = cache->k_sink; A.v_sink = cache->v_sink; A.n_sink = cache->n_sink;
  A.ticket = (int32_t*)scratch;
  A.q = q; A.out = out; A.ws = (float*)(scratch + STATIC_TICKET_BYTES);
  A.B = cache->B; A.Hkv = cache->Hkv; A.Hq = Hq; A.g = g; A.max_chunks = cache->max_chunks;
  A.cluster = sp.cluster; A.nclus = sp.nclus; A.splits = sp.cluster * sp.nclus;
  A.q_scale = sm_scale * 1.4426950408889634f;
  A.rotate_k = p->rotate_k; A.rotate_v = p->rotate_v; A.out_dtype = p->out_dtype;
  A.n_q = 1; A.tpc = 1; A.k_blk = nullptr; A.v_blk = nullptr; A.partial = 0;
  const cudaError_t e = launch_decode(p, A, s);
  return e == cudaSuccess ? KVARN_OK : KVARN_CUDA;
}

int kvarn_merge_partials(const float* parts, int32_t n_parts, int64_t n_rows, void* out, int32_t out_dtype,
                         void* stream) {
  if (!parts || !out || n_parts < 1 || n_rows < 0) return KVARN_INVALID_ARG;
  if (out_dtype != KVARN_BF16 && out_dtype != KVARN_F32) return KVARN_UNSUPPORTED;
  if (!aligned16(parts) || !aligned16(out)) return KVARN_MISALIGNED;
  if (n_rows == 0) return KVARN_OK;
  merge_partials_kernel<<<(unsigned)n_rows, 128, 0, (cudaStream_t)stream>>>(parts, n_parts, n_rows, out, out_dtype);
  return last_cuda();
}

// Multi-token read path (Fig. 4): the same kernel, the (query token, head)
// pairs that share a KV head are its MMA columns, 8 per CTA; blockIdx.z walks the block in groups of
// tpc = 8 / g tokens.  Split-K only through one thread-block cluster (no workspace merge).
int kvarn_block_attention(const kvarn_params* p, const kvarn_cache* cache, const void* q,
                          const void* k_blk, const void* v_blk, int32_t n_q, int32_t Hq,
                          float sm_scale, void* out, void* stream) {
  int st = check_params(p);
  if (st) return st;
  if ((st = check_cache(cache))) return st;
  if (!q || !out || !k_blk || !v_blk || Hq <= 0 || (Hq % cache->Hkv) != 0 || n_q < 1) return KVARN_INVALID_ARG;
  const int g = Hq / cache->Hkv;
  if (g > 8 || (g & (g - 1)) || n_q > G) return KVARN_UNSUPPORTED;
  if (!aligned16(q) || !aligned16(out) || !aligned16(k_blk) || !aligned16(v_blk)) return KVARN_MISALIGNED;
  DecodeArgs A{};
  A.k_records = (const uint8_t*)cache->k_records; A.v_records = (const uint8_t*)cache->v_records;
  A.k_resid = cache->k_resid; A.v_resid = cache->v_resid; A.seq_lens = cache->seq_lens;
  A.k_sink = cache->k_sink; A.v_sink = cache->v_sink; A.n_sink = cache->n_sink;
  A.ticket = cache->decode_ticket;   // unused: nclus = 1
  A.q = q; A.out = out; A.ws = nullptr;
  A.B = cache->B; A.Hkv = cache->Hkv; A.Hq = Hq; A.g = g; A.max_chunks = cache->max_chunks;
  A.n_q = n_q; A.k_blk = k_blk; A.v_blk = v_blk;
  A.tpc = n_q * g <= 4 ? n_q : (8 / g < n_q ? 8 / g : n_q);
  const int nz = (n_q + A.tpc - 1) / A.tpc;
  int want = p->splits > 0 ? p->splits : decode_slots(p, A.tpc * g) / (cache->B * cache->Hkv * nz);
  if (want > KVARN_MAX_CLUSTER) want = KVARN_MAX_CLUSTER;
  if (want > cache->max_chunks) want = cache->max_chunks;
  if (want < 1) want = 1;
  A.cluster = want; A.nclus = 1; A.splits = want;
  A.q_scale = sm_scale * 1.4426950408889634f;
  A.rotate_k = p->rotate_k; A.rotate_v = p->rotate_v; A.out_dtype = p->out_dtype;
  const cudaError_t e = launch_decode(p, A, (cudaStream_t)stream);
  return e == cudaSuccess ? KVARN_OK : KVARN_CUDA;
}

// Dense form of kvarn_block_attention for blocks with many query rows per KV head (tcgen05 + TMEM; kvarn_block_dense.cuh):
// packed chunks and raw windows by block_dense_kernel, its partial sets merged by merge_partials_kernel.
static int dense_splits(int B, int Hkv, int n_tiles, int max_chunks) {
  int sms = 148;
  const int dev = current_device();
  if (dev >= 0 && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) { cudaGetLastError(); sms = 148; }
#ifdef KVARN_DENSE_SPLITS_ENV
  if (const char* e = getenv("KVARN_DENSE_SPLITS")) { const int v = atoi(e); if (v > 0) return v > 32 ? 32 : v; }
#endif
  // One CTA per SM (210 KB of shared memory, 512 TMEM columns), so the CTAs run in waves of `sms`.  Cost of a plan in
  // chunk-times: waves x (chunks per CTA + the fixed cost of a CTA: prologue, pipeline fill and drain, epilogue), plus
  // the merge launch when a row tile is spread over several CTAs -- fitted to measured splits 1..16 on the 64k-context
  // cache.  Few units: the chunks spread over the idle SMs; many units: the split that fills the
  // last wave (512 CTAs on 148 SMs: 2 per row tile make 7 full waves of 256 chunks instead of 4 of 512).
  const long long ctas = (long long)B * Hkv * n_tiles;
  int best = 1;
  long long best_cost = -1;
  for (int s = 1; s <= 32; ++s) {
    const int per = (max_chunks + s - 1) / s;
    if (s > 1 && per < 4) break;                 // at least 4 chunks per CTA
    const long long waves = (ctas * s + sms - 1) / sms;
    const long long cost = waves * (per + KVARN_DENSE_CTA_COST) + (s > 1 ? KVARN_DENSE_MERGE_COST : 0);
    if (best_cost < 0 || cost < best_cost) { best_cost = cost; best = s; }
  }
  return best;
}

size_t kvarn_block_dense_workspace_bytes(const kvarn_params* p, int32_t B, int32_t Hq, int32_t Hkv, int32_t n_q,
                                         int32_t max_chunks) {
  if (!p || B <= 0 || Hq <= 0 || Hkv <= 0 || n_q <= 0 || (Hq % Hkv) != 0) return 0;
  const int g = Hq / Hkv, n_tiles = (n_q * g + 127) / 128;
  return (size_t)dense_splits(B, Hkv, n_tiles, max_chunks) * B * n_q * Hq * PART_STRIDE * sizeof(float);   // touched only when > 1 split
}

int kvarn_block_attention_dense(const kvarn_params* p, const kvarn_cache* cache, const void* q,
                                const void* k_blk, const void* v_blk, int32_t n_q, int32_t Hq,
                                float sm_scale, void* out, void* ws, size_t ws_bytes, void* stream) {
  int st = check_params(p);
  if (st) return st;
  if ((st = check_cache(cache))) return st;
  if (!q || !out || !k_blk || !v_blk || !ws || Hq <= 0 || (Hq % cache->Hkv) != 0 || n_q < 1) return KVARN_INVALID_ARG;
  const int g = Hq / cache->Hkv;
  if (g > 8 || (g & (g - 1)) || n_q > G) return KVARN_UNSUPPORTED;
  if (!aligned16(q) || !aligned16(out) || !aligned16(k_blk) || !aligned16(v_blk) || !aligned16(ws)) return KVARN_MISALIGNED;
  if (ws_bytes < kvarn_block_dense_workspace_bytes(p, cache->B, Hq, cache->Hkv, n_q, cache->max_chunks)) return KVARN_WORKSPACE_TOO_SMALL;
  cudaStream_t s = (cudaStream_t)stream;
  const bool f32 = p->in_dtype == KVARN_F32;
  const long long n_rows = (long long)cache->B * n_q * Hq;
  DenseArgs E{};
  E.k_records = (const uint8_t*)cache->k_records; E.v_records = (const uint8_t*)cache->v_records; E.seq_lens = cache->seq_lens;
  E.q = q; E.parts = (float*)ws; E.out = out; E.out_dtype = p->out_dtype;
  E.k_resid = cache->k_resid; E.v_resid = cache->v_resid; E.k_sink = cache->k_sink; E.v_sink = cache->v_sink;
  E.k_blk = k_blk; E.v_blk = v_blk;
  E.B = cache->B; E.Hkv = cache->Hkv; E.Hq = Hq; E.g = g; E.max_chunks = cache->max_chunks; E.n_sink = cache->n_sink; E.n_q = n_q;
  E.n_tiles = (n_q * g + 127) / 128;
  E.splits = dense_splits(cache->B, cache->Hkv, E.n_tiles, cache->max_chunks);
  E.q_scale = sm_scale * 1.4426950408889634f; E.rotate_k = p->rotate_k; E.rotate_v = p->rotate_v;
  {
    const dim3 grid((unsigned)(cache->B * cache->Hkv * E.n_tiles), (unsigned)E.splits);
    cudaError_t e;
    if (p->bits == 2) {
      if (f32) { e = ensure_smem_optin<block_dense_kernel<2, float>>((int)sizeof(DenseSmem<2>), true);
                 if (e == cudaSuccess) block_dense_kernel<2, float><<<grid, DENSE_THREADS, sizeof(DenseSmem<2>), s>>>(E); }
      else { e = ensure_smem_optin<block_dense_kernel<2, __nv_bfloat16>>((int)sizeof(DenseSmem<2>), true);
             if (e == cudaSuccess) block_dense_kernel<2, __nv_bfloat16><<<grid, DENSE_THREADS, sizeof(DenseSmem<2>), s>>>(E); }
    } else {
      if (f32) { e = ensure_smem_optin<block_dense_kernel<4, float>>((int)sizeof(DenseSmem<4>), true);
                 if (e == cudaSuccess) block_dense_kernel<4, float><<<grid, DENSE_THREADS, sizeof(DenseSmem<4>), s>>>(E); }
      else { e = ensure_smem_optin<block_dense_kernel<4, __nv_bfloat16>>((int)sizeof(DenseSmem<4>), true);
             if (e == cudaSuccess) block_dense_kernel<4, __nv_bfloat16><<<grid, DENSE_THREADS, sizeof(DenseSmem<4>), s>>>(E); }
    }
    if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) return KVARN_CUDA;
  }
  // (the raw windows -- sink, residual, the block's own causal tokens -- ran inside the same kernel as extra chunks)
  if (E.splits > 1) merge_partials_kernel<<<(unsigned)n_rows, 128, 0, s>>>((const float*)ws, E.splits, n_rows, out, p->out_dtype);
  return last_cuda();
}

int kvarn_rope_hadamard(const void* x, const float* cos_tab, const float* sin_tab, void* y, int64_t n_tok,
                        int32_t n_heads, int32_t dtype, int32_t rotate, void* stream) {
  if (n_tok == 0) return KVARN_OK;
  if (!x || !y || n_tok < 0 || n_heads <= 0 || (!cos_tab) != (!sin_tab)) return KVARN_INVALID_ARG;
  if (dtype != KVARN_BF16 && dtype != KVARN_F32) return KVARN_UNSUPPORTED;
  if (!aligned16(x) || !aligned16(y) || !aligned16(cos_tab) || !aligned16(sin_tab)) return KVARN_MISALIGNED;
  const long long n_groups = (long long)n_tok * n_heads;
  if (n_groups == 0) return KVARN_OK;
  const unsigned grid = (unsigned)((n_groups + 8 * ROT_GPW - 1) / (8 * ROT_GPW));
  cudaStream_t s = (cudaStream_t)stream;
  if (dtype == KVARN_F32)
    rope_hadamard_kernel<float><<<grid, 256, 0, s>>>((const float*)x, cos_tab, sin_tab, (float*)y, n_groups, n_heads, rotate);
  else
    rope_hadamard_kernel<__nv_bfloat16><<<grid, 256, 0, s>>>((const __nv_bfloat16*)x, cos_tab, sin_tab, (__nv_bfloat16*)y,
                                                          n_groups, n_heads, rotate);
  return last_cuda();
}

int kvarn_hadamard_rows(const void* x, void* y, int64_t n_groups, int32_t dtype, void* stream) {
  return kvarn_rope_hadamard(x, nullptr, nullptr, y, n_groups, 1, dtype, 1, stream);
}

int kvarn_hadamard_row_groups(const void* w, void* out, int64_t n_rows, int64_t n_cols, int32_t dtype, void* stream) {
  if (!w || !out || n_rows < 0 || n_cols < 0 || (n_rows % G) != 0) return KVARN_INVALID_ARG;
  if (dtype != KVARN_BF16 && dtype != KVARN_F32) return KVARN_UNSUPPORTED;
  if (n_rows == 0 || n_cols == 0) return KVARN_OK;
  if (n_rows / G > 65535) return KVARN_UNSUPPORTED;
  const dim3 grid((unsigned)((n_cols + 31) / 32), (unsigned)(n_rows / G));
  cudaStream_t s = (cudaStream_t)stream;
  if (dtype == KVARN_F32) hadamard_row_groups_kernel<float><<<grid, 128, 0, s>>>((const float*)w, (float*)out, n_cols);
  else hadamard_row_groups_kernel<__nv_bfloat16><<<grid, 128, 0, s>>>((const __nv_bfloat16*)w, (__nv_bfloat16*)out, n_cols);
  return last_cuda();
}

int kvarn_quantize_chunk_host(const kvarn_params* p, const void* k_host, const void* v_host,
                              int64_t n_tiles, void* dev_in_k, void* dev_in_v, void* dev_rec_k,
                              void* dev_rec_v, void* k_rec_host, void* v_rec_host, void* stream) {
  int st = check_params(p);
  if (st) return st;
  if (!k_host || !v_host || !dev_in_k || !dev_in_v || !dev_rec_k || !dev_rec_v || n_tiles < 0) return KVARN_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  const size_t esz = p->in_dtype == KVARN_F32 ? 4 : 2;
  const size_t in_bytes = (size_t)n_tiles * G * D * esz, rec_b = (size_t)n_tiles * record_bytes(p->bits);
  if (cudaMemcpyAsync(dev_in_k, k_host, in_bytes, cudaMemcpyHostToDevice, s) != cudaSuccess) return KVARN_CUDA;
  if (cudaMemcpyAsync(dev_in_v, v_host, in_bytes, cudaMemcpyHostToDevice, s) != cudaSuccess) return KVARN_CUDA;
  st = kvarn_quantize_chunk(p, dev_in_k, dev_in_v, n_tiles, (int64_t)G * D, D, dev_rec_k, dev_rec_v,
                            record_bytes(p->bits), nullptr, stream);
  if (st) return st;
  if (k_rec_host && cudaMemcpyAsync(k_rec_host, dev_rec_k, rec_b, cudaMemcpyDeviceToHost, s) != cudaSuccess) return KVARN_CUDA;
  if (v_rec_host && cudaMemcpyAsync(v_rec_host, dev_rec_v, rec_b, cudaMemcpyDeviceToHost, s) != cudaSuccess) return KVARN_CUDA;
  return KVARN_OK;
}

int kvarn_decode_attention_host(const kvarn_params* p, const kvarn_cache* cache,
                                const void* q_host, int32_t Hq, float sm_scale, void* out_host,
                                void* dev_q, void* dev_out, void* ws, size_t ws_bytes,
                                void* stream) {
  int st = check_params(p);
  if (st) return st;
  if (!cache || !q_host || !out_host || !dev_q || !dev_out || Hq <= 0) return KVARN_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  const size_t n = (size_t)cache->B * Hq * D;
  const size_t qb = n * (p->in_dtype == KVARN_F32 ? 4 : 2), ob = n * (p->out_dtype == KVARN_F32 ? 4 : 2);
  if (cudaMemcpyAsync(dev_q, q_host, qb, cudaMemcpyHostToDevice, s) != cudaSuccess) return KVARN_CUDA;
  st = kvarn_decode_attention(p, cache, dev_q, Hq, sm_scale, dev_out, ws, ws_bytes, stream);
  if (st) return st;
  if (cudaMemcpyAsync(out_host, dev_out, ob, cudaMemcpyDeviceToHost, s) != cudaSuccess) return KVARN_CUDA;
  return KVARN_OK;
}

int kvarn_unpack_record_host(const kvarn_params* p, int32_t kind, const void* record,
                             uint8_t* codes, float* s1, float* s2, float* z) {
  if (!p || !record || !codes || !s1 || !s2 || !z) return KVARN_INVALID_ARG;
  if (p->bits != 2 && p->bits != 4) return KVARN_UNSUPPORTED;
  if (kind != KVARN_KIND_K && kind != KVARN_KIND_V) return KVARN_INVALID_ARG;
  const int bits = p->bits, lv = (1 << bits) - 1, per_byte = 8 / bits, rowb = row_bytes(bits);
  const uint8_t* r = (const uint8_t*)record;
  (void)rowb;
  for (int row = 0; row < 128; ++row)
    for (int e = 0; e < 128; ++e) {
      const int slot = (kind == KVARN_KIND_K) ? slot_of_token(bits, row) : row;
      const uint8_t byte = r[code_off(bits, slot, e / per_byte)];
      const uint8_t code = (byte >> (bits * (e % per_byte))) & lv;
      if (kind == KVARN_KIND_K) codes[row * 128 + e] = code;   // row = token, e = channel
      else codes[e * 128 + row] = code;                        // row = channel, e = token
    }
  for (int i = 0; i < 128; ++i) {
    // K: s1, z per channel in B-operand builder order, s2 per token in row-slot order;
    // V: s1, z per token in row-slot order, s2 per channel in natural order
    const int gi = (kind == KVARN_KIND_K) ? kaux_of_elem(bits, i) : slot_of_token(bits, i);
    const int si = (kind == KVARN_KIND_K) ? slot_of_token(bits, i) : i;
    s1[i] = e4m3_to_f32(r[s1_off(bits) + gi]);
    s2[i] = e4m3_to_f32(r[s2_off(bits) + si]);
    uint16_t zb;
    memcpy(&zb, r + z_off(bits) + 2 * gi, 2);
    z[i] = f16_bits_to_f32(zb);
  }
  return KVARN_OK;
}

int kvarn_pack_record_host(const kvarn_params* p, int32_t kind, const uint8_t* codes,
                           const float* s1, const float* s2, const float* z, void* record) {
  if (!p || !record || !codes || !s1 || !s2 || !z) return KVARN_INVALID_ARG;
  if (p->bits != 2 && p->bits != 4) return KVARN_UNSUPPORTED;
  if (kind != KVARN_KIND_K && kind != KVARN_KIND_V) return KVARN_INVALID_ARG;
  const int bits = p->bits, lv = (1 << bits) - 1, per_byte = 8 / bits, rowb = row_bytes(bits);
  uint8_t* r = (uint8_t*)record;
  memset(r, 0, record_bytes(bits));
  (void)rowb;
  for (int row = 0; row < 128; ++row)
    for (int e = 0; e < 128; ++e) {
      const uint8_t code = (kind == KVARN_KIND_K ? codes[row * 128 + e] : codes[e * 128 + row]) & lv;
      const int slot = (kind == KVARN_KIND_K) ? slot_of_token(bits, row) : row;
      r[code_off(bits, slot, e / per_byte)] |= (uint8_t)(code << (bits * (e % per_byte)));
    }
  for (int i = 0; i < 128; ++i) {
    const int gi = (kind == KVARN_KIND_K) ? kaux_of_elem(bits, i) : slot_of_token(bits, i);
    const int si = (kind == KVARN_KIND_K) ? slot_of_token(bits, i) : i;
    r[s1_off(bits) + gi] = f32_to_e4m3(s1[i]);
    r[s2_off(bits) + si] = f32_to_e4m3(s2[i]);
    const uint16_t zb = f32_to_f16_bits(z[i]);
    memcpy(r + z_off(bits) + 2 * gi, &zb, 2);
  }
  return KVARN_OK;
}

}  // extern "C"

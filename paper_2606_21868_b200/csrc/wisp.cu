// wisp.cu -- context, C ABI (include/wisp.h) and launch orchestration of libwisp (sm_100a).
// Host code only enqueues work; every step of the hot path (router, residency, fetch, FFN, combine)
// runs in the kernels of router.cuh / residency.cuh / fetch.cuh / decode_*.cuh / ffn_prefill*.cuh.
#include <algorithm>
#include <cstdio>
#include <cstring>
#include <map>
#include <string>
#include <thread>
#include <vector>

#include "common.cuh"
#include "decode_kernels.cuh"
#include "fetch.cuh"
#include "ffn_prefill.cuh"
#include "ffn_prefill_mma.cuh"
#include "mvwsa.h"
#include "prefetch.cuh"
#include "residency.cuh"
#include "router.cuh"

using namespace wisp;

static_assert(sizeof(wisp_config) == 72 && sizeof(wisp_trace_event) == 32, "C ABI struct layout (tests/test_library_abi.py mirrors it)");

struct wisp_ctx {
  wisp_config cfg{};
  u64 budget = 0;
  size_t elem = 0, Me = 0, a_bytes = 0, blob_elems = 0;   // elem: bytes per hidden-state / router element
  size_t welem = 0;                // bytes per expert-weight element (1 for WISP_FP8_E4M3)
  bool f8 = false;
  size_t s13_off = 0, s2_off = 0;  // fp8: byte offsets of the block scales inside a blob (S13, then S2 transposed)
  int C = 0;
  u64 kappa = 0, kv_reserved = 0, kv_peak = 0;
  u64 resize_count = 0, failed_resize = 0;
  int num_sms = 0;

  char* arena = nullptr;
  std::vector<void*> master;       // pinned, mapped; one allocation per layer, blobs in the tiled in-slot layout
  std::vector<char> registered;
  char* router_w = nullptr;        // device [L][E][d]   (prefill router GEMM)
  char* router_wt = nullptr;       // device [L][d][E]   (decode: 16-column slices of the hidden state)
  float* router_bias = nullptr;    // device [L][E]

  // per-layer residency state (device), each [L][...]
  int *pi = nullptr, *pi_inv = nullptr;
  u64 *tau = nullptr, *freq = nullptr, *scal = nullptr, *last_pos = nullptr, *hist = nullptr;

  // per-forward scratch (device)
  float* logits = nullptr;         // [maxT][E]
  int* ids = nullptr;              // [L][maxT*k]
  float* topw = nullptr;           // [L][maxT*k]
  std::vector<int> last_T;
  int last_layer = -1;
  int* plan_mem = nullptr;
  PlanPtrs plan{};
  HostPlan* host_plan = nullptr;   // mapped pinned
  char* act_T = nullptr;           // [maxT*k][d_ff] model dtype (prefill)
  float* ystage = nullptr;         // [maxT*k][d] (prefill)
  char* xbuf[2] = {nullptr, nullptr};
  char* ybuf = nullptr;
  int* dbg_ids = nullptr;
  size_t dbg_ids_cap = 0;
  int* moves = nullptr;            // [2*E] + n_moves
  int* bad_slots = nullptr;        // [E]

  wisp_trace_event* trace = nullptr;
  u64* trace_ctr = nullptr;        // device [2]
  u64 trace_cap = 0;
  int trace_on = 0;
  int wave_order = WISP_WAVES_ASCENDING;   // G25
  int track = 0;
  std::vector<double> host_hist;

  cudaStream_t copy_stream = nullptr;
  cudaEvent_t ev_plan = nullptr, ev_compute = nullptr, ev_copy = nullptr;
  int timing_level = 0;            // 0 off, 1 miss path only, 2 every kernel class
  struct TimedSpan { cudaEvent_t a, b; int cls; };
  std::vector<TimedSpan> timing_pool;
  size_t timing_used = 0;
  double class_ms[WISP_N_KERNEL_CLASSES] = {};
  u64 class_n[WISP_N_KERNEL_CLASSES] = {};
  u64 launches = 0;
  std::map<int, u64> graph_nodes;

  std::map<int, cudaGraphExec_t> graphs;   // decode-sized stacks only (n_tokens <= kDecodeMaxTokens)
  int grid_fetch = 0;
  // decode path (decode_*.cuh)
  DecodeGeom dgeom[2]{};             // [0]: calls of at most 2 tokens, [1]: 3..8 tokens (larger work units: fewer chunk partials)
  float* partial = nullptr;          // chunk partials P [pair position][NC][d]
  long long* zfix = nullptr;         // [2][kZfixCopies][kDecodeMaxTokens][E] int64 logit accumulators (zero between launches)
  unsigned* dsync = nullptr;         // [0] grid barrier counter, [1..2] unit tickets
  const char** d_masters = nullptr;  // device [L]: mapped master pointers
  int* host_err = nullptr;           // mapped pinned flag: a grid barrier of the fused kernel timed out
  int* dev_err = nullptr;            // its device alias
  u64* phase_ns = nullptr;           // device [kDecPhases + 2]
  size_t fused_smem = 0, ffn_smem = 0;   // dynamic shared memory available to the fused / split ffn kernel on this device
  int persist_enabled = 1;
  // static layer-offload comparison arm (WISP_FETCH_STATIC): resident layers [0, static_pinned) at arena + l*E*M_e, then a
  // two-layer bounce region; every other layer is streamed from its master on every forward
  int static_pinned = 0;
  char* bounce[2] = {nullptr, nullptr};
  cudaEvent_t ev_buf_free[2] = {nullptr, nullptr}, ev_buf_ready[2] = {nullptr, nullptr};
  bool buf_used[2] = {false, false};
  u64 static_streamed = 0;         // bytes copied into the bounce region so far
  bool is_static() const { return cfg.fetch == WISP_FETCH_STATIC; }
  // speculative prefetch (prefetch.cuh; wisp_set_prefetch)
  int pf_n = 0, pf_window = 1;
  double pf_gpow[kMaxWindow + 1] = {};
  unsigned *pf_A = nullptr, *pf_row = nullptr;
  int *pf_rlist = nullptr, *pf_rcount = nullptr, *pf_copy = nullptr;   // copy lists [L][1 + 2 * kMaxPrefetch]
  cudaStream_t pf_stream = nullptr;
  std::vector<cudaEvent_t> ev_pred, ev_copied;
  std::vector<char> pf_pending;
  // tcgen05 prefill path (ffn_prefill_mma.cuh): TMA tensor maps over the arena / the B-operand buffers
  bool mma_ok = false;
  CUtensorMap tm_gu{}, tm_dn{}, tm_xg{}, tm_act{}, tm_rw{};
  void* encode_fn = nullptr;         // cuTensorMapEncodeTiled (per-call map over the caller's hidden states)
  char* xg = nullptr;                // [maxT*k][d] gathered token rows (bf16)
  int* mma_work = nullptr;           // work list of the current wave: (entry, first pair) items + count
  u64 fused_layers_timed = 0;
  bool use_fused(int T_) const {
    return persist_enabled && cfg.fetch == WISP_FETCH_FUSED && T_ <= kDecodeMaxTokens && cfg.n_experts <= kPersistMaxExperts;
  }
  std::string err;
};

namespace {

const char* kVersion = "libwisp 0.1 (sm_100a; router/residency/fetch/ffn kernels; build " __DATE__ ")";

int fail(wisp_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg;
  return code;
}

#define CK(call)                                                                                   \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess)                                                                         \
      return fail(ctx, e_ == cudaErrorMemoryAllocation ? WISP_ENOMEM : WISP_ECUDA,                 \
                  std::string(#call) + ": " + cudaGetErrorString(e_));                             \
  } while (0)

LayerState layer_state(wisp_ctx* c, int l) {
  const size_t E = c->cfg.n_experts;
  LayerState s;
  s.pi = c->pi + l * E;
  s.pi_inv = c->pi_inv + l * E;
  s.tau = c->tau + l * E;
  s.freq = c->freq + l * E;
  s.scal = c->scal + l * 8;
  s.last_pos = c->last_pos + l * E;
  s.hist = c->hist + l * (E + 2);
  return s;
}

void drop_graphs(wisp_ctx* c) {
  for (auto& g : c->graphs) cudaGraphExecDestroy(g.second);
  c->graphs.clear();
}

void harvest_timing(wisp_ctx* c, bool all) {
  size_t keep = 0;
  for (size_t i = 0; i < c->timing_used; ++i) {
    auto& p = c->timing_pool[i];
    if (all) cudaEventSynchronize(p.b);
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, p.a, p.b) == cudaSuccess) { c->class_ms[p.cls] += ms; c->class_n[p.cls] += 1; }
    else std::swap(c->timing_pool[keep++], p);
  }
  c->timing_used = keep;
}

// RAII span around one launch: counts it, and when timing is on brackets it with CUDA events on `st`.
struct Span {
  wisp_ctx* c;
  cudaStream_t st;
  cudaEvent_t b = nullptr;
  Span(wisp_ctx* c_, int cls, cudaStream_t st_, bool is_kernel = true) : c(c_), st(st_) {
    if (is_kernel) ++c->launches;
    if (c->timing_level == 0 || (c->timing_level == 1 && cls != WISP_K_FETCH)) return;
    if (c->timing_used == c->timing_pool.size()) {
      harvest_timing(c, false);
      if (c->timing_used == c->timing_pool.size()) {
        if (c->timing_pool.size() >= 8192) harvest_timing(c, true);
        else {
          cudaEvent_t x, y;
          if (cudaEventCreate(&x) != cudaSuccess || cudaEventCreate(&y) != cudaSuccess) return;
          c->timing_pool.push_back({x, y, 0});
        }
      }
    }
    auto& p = c->timing_pool[c->timing_used++];
    p.cls = cls;
    cudaEventRecord(p.a, st);
    b = p.b;
  }
  ~Span() { if (b) cudaEventRecord(b, st); }
};

// ---- TMA tensor maps (tcgen05 prefill path) ----
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

bool make_tmap(EncodeTiledFn fn, CUtensorMap* tm, void* base, int rank, const cuuint64_t* dims, const cuuint64_t* strides_bytes,
               const cuuint32_t* box, bool swizzle128) {
  cuuint32_t estr[4] = {1, 1, 1, 1};
  return fn(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, (cuuint32_t)rank, base, dims, strides_bytes, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, swizzle128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <typename T>
int launch_router(wisp_ctx* ctx, int layer, const void* x, int T_, cudaStream_t st) {
  const auto& cfg = ctx->cfg;
  const int E = cfg.n_experts, d = cfg.d_model, k = cfg.top_k;
  const T* wr = reinterpret_cast<const T*>(ctx->router_w) + (size_t)layer * E * d;
  dim3 g((E + 7) / 8, (T_ + kRouterTokTile - 1) / kRouterTokTile);
  if (ctx->mma_ok && T_ > kDecodeMaxTokens && E % kMmaM == 0 && sizeof(T) == 2) {
    // prefill: the router is a [T x d] x [d x E] GEMM -> same tcgen05 kernel (MODE 2), B operand = the caller's rows
    CUtensorMap tm_x;
    const cuuint64_t dims[2] = {(cuuint64_t)d, (cuuint64_t)T_}, str[1] = {(cuuint64_t)d * 2};
    const int b_rows = 32;
    const cuuint32_t box2[2] = {kMmaBK, (cuuint32_t)b_rows};
    if (!make_tmap(reinterpret_cast<EncodeTiledFn>(ctx->encode_fn), &tm_x, const_cast<void*>(x), 2, dims, str, box2, true))
      return fail(ctx, WISP_ECUDA, "tensor map over the hidden states failed (16-byte aligned rows required)");
    MmaArgs m{};
    m.L = cfg.n_layers; m.layer = layer; m.d = d; m.dff = cfg.d_ff; m.k = k;
    m.z = ctx->logits; m.bias = ctx->router_bias + (size_t)layer * E; m.n_tokens = T_; m.E = E; m.b_rows = b_rows;
    Span sp(ctx, WISP_K_ROUTER, st);
    const int ns = 6;
    prefill_mma_kernel<2><<<ctx->num_sms, kMmaThreads, ns * 2 * kMmaTileBytes + 1024, st>>>(ctx->tm_rw, tm_x, m, nullptr, nullptr, ns);
  } else {
    Span sp(ctx, WISP_K_ROUTER, st);
    router_logits_kernel<T><<<g, 256, 0, st>>>(reinterpret_cast<const T*>(x), wr, ctx->router_bias + (size_t)layer * E,
                                               ctx->logits, T_, E, d);
  }
  const size_t off = (size_t)layer * cfg.max_tokens * k;
  {
    Span sp(ctx, WISP_K_TOPK, st);
    if (E <= 256) topk_softmax_kernel<8><<<(T_ + 3) / 4, 128, 0, st>>>(ctx->logits, ctx->ids + off, ctx->topw + off, T_, E, k);
    else topk_softmax_kernel<kMaxExperts / 32><<<(T_ + 3) / 4, 128, 0, st>>>(ctx->logits, ctx->ids + off, ctx->topw + off, T_, E, k);
  }
  CK(cudaGetLastError());
  return WISP_OK;
}

int launch_plan(wisp_ctx* ctx, int layer, const int* ids, int n_pairs, bool want_host, cudaStream_t st) {
  PlanArgs a;
  a.ids = ids;
  a.n_pairs = n_pairs;
  a.E = ctx->cfg.n_experts;
  a.C = ctx->C;
  a.policy = ctx->cfg.policy;
  a.layer = layer;
  a.st = layer_state(ctx, layer);
  a.plan = ctx->plan;
  a.host_plan = want_host ? ctx->host_plan : nullptr;
  a.trace = ctx->trace;
  a.trace_ctr = ctx->trace_ctr;
  a.trace_cap = ctx->trace_cap;
  a.trace_on = ctx->trace_on;
  a.wave_order = ctx->wave_order;
  a.track = ctx->track;
  a.build_pairs = n_pairs <= 256;
  {
    Span sp(ctx, WISP_K_RESIDENCY, st);
    residency_plan_kernel<<<1, kPlanThreads, 0, st>>>(a);
  }
  if (!a.build_pairs) {
    Span sp(ctx, WISP_K_RESIDENCY, st);
    group_pairs_kernel<<<a.E, kGroupThreads, 0, st>>>(ids, n_pairs, ctx->plan);
  }
  CK(cudaGetLastError());
  return WISP_OK;
}

// Miss path for one wave.  ZEROCOPY: one kernel on the compute stream.  MEMCPY: host-read miss list ->
// cudaMemcpyAsync on the copy stream, fenced both ways with events.
int fetch_wave(wisp_ctx* ctx, int layer, int wave, bool host_known, cudaStream_t st) {
  const auto& cfg = ctx->cfg;
  const size_t blob_vec = ctx->Me / 16;
  if (!host_known) {
    {
      Span sp(ctx, WISP_K_FETCH, st);
      fetch_zerocopy_kernel<<<ctx->grid_fetch, kFetchThreads, 0, st>>>(
          ctx->plan, wave, ctx->C, reinterpret_cast<const uint4*>(ctx->master[layer]),
          reinterpret_cast<uint4*>(ctx->arena), blob_vec, cfg.n_layers, layer);
    }
    CK(cudaGetLastError());
    return WISP_OK;
  }
  const HostPlan* hp = ctx->host_plan;
  const int lo = wave * ctx->C, hi = std::min(hp->n_ref, lo + ctx->C);
  bool any = false;
  for (int i = lo; i < hi; ++i) any |= hp->entry_miss[i] != 0;
  if (!any) return WISP_OK;
  CK(cudaEventRecord(ctx->ev_compute, st));
  CK(cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_compute, 0));
  {
    Span sp(ctx, WISP_K_FETCH, ctx->copy_stream, /*is_kernel=*/false);
    for (int i = lo; i < hi; ++i) {
      if (!hp->entry_miss[i]) continue;
      const char* src = static_cast<const char*>(ctx->master[layer]) + (size_t)hp->entry_expert[i] * ctx->Me;
      char* dst = ctx->arena + ((size_t)hp->entry_slot[i] * cfg.n_layers + layer) * ctx->Me;
      CK(cudaMemcpyAsync(dst, src, ctx->Me, cudaMemcpyHostToDevice, ctx->copy_stream));
    }
  }
  CK(cudaEventRecord(ctx->ev_copy, ctx->copy_stream));
  CK(cudaStreamWaitEvent(st, ctx->ev_copy, 0));
  return WISP_OK;
}

// ---- decode path (decode_*.cuh) --------------------------------------------------------------------------------
// Geometry of the fused FFN stream: slab = the largest multiple-of-256 divisor of d whose 8-row part fits 32 KiB.
DecodeGeom make_decode_geom(int d, int dff, size_t elem, int rows_unit, bool f8 = false) {
  DecodeGeom g{};
  g.d = d; g.dff = dff; g.elem = (int)elem; g.kc = (int)(16 / elem);
  int m = (int)(kDecMaxPartBytes / (8 * elem)) / 256;
  if (f8) m = std::min(m, kDecMaxSteps * 128 / 256);          // a warp's range of a slab is at most kDecMaxSteps cores
  const int q = d / 256;
  while (q % m) --m;
  g.slab = 256 * m;
  g.n_slab = d / g.slab;
  g.rows_unit = rows_unit;
  g.n_sb = rows_unit / 8;
  g.sub_bytes = 8 * g.slab * (int)elem;
  g.merge = f8 && g.n_slab == 1 && g.n_sb == 2 && g.n_sb * g.sub_bytes <= kDecMaxPartBytes ? 1 : 0;   // (the merged down pass feeds 16 k slots)
  g.part_bytes = g.sub_bytes * (g.merge ? g.n_sb : 1);
  g.n_chunks = dff / rows_unit;
  g.parts_unit = 3 * g.n_sb * g.n_slab;
  g.steps = g.slab / 128;
  g.down_pieces = f8 ? 1 : 8 / g.kc;
  g.up_off = (unsigned long long)dff * d * elem;
  g.down_off = 2 * g.up_off;
  g.group_bytes = 8ull * d * elem;
  g.f8 = f8 ? 1 : 0;
  g.act_elem = f8 ? 2 : (int)elem;
  g.scale_bytes = f8 ? 4 * (g.slab / 128) : 0;
  g.slot_bytes = g.part_bytes + g.scale_bytes;
  g.s13_off = 3ull * d * dff * elem;
  g.s2_off = g.s13_off + 4ull * (2 * dff / 128) * (d / 128);
  return g;
}

struct DecodeSmem { int n_slots, xs_pitch, pre_off, ring_off; size_t bytes; };
// Shared-memory carve-up of a decode CTA: [hidden states, rows padded by 16 B][staged router-weight slice (fused kernel)]
// [ring of n_slots parts].
int decode_smem(wisp_ctx* ctx, const DecodeGeom& g, int T_, size_t avail, bool fused, DecodeSmem* out) {
  out->xs_pitch = g.d + 16 / g.act_elem;
  out->pre_off = (int)(((size_t)T_ * out->xs_pitch * g.act_elem + 127) & ~(size_t)127) * (g.f8 ? 2 : 1);   // fp8: + the f16 copy
  const size_t pre = fused ? (((size_t)ctx->cfg.n_experts * sizeof(float) + 127) & ~(size_t)127) +
                                 (((size_t)kSliceCols * ctx->cfg.n_experts * g.act_elem + 127) & ~(size_t)127) : 0;
  out->ring_off = out->pre_off + (int)pre;
  if ((size_t)out->ring_off + 2 * (size_t)g.slot_bytes > avail) return fail(ctx, WISP_EINVAL, "decode kernel: shared memory too small for this shape");
  int n = (int)std::min<size_t>(kDecMaxSlots, (avail - out->ring_off) / g.slot_bytes);
  if (ctx->cfg.ring_stages > 0) n = std::min(n, std::max(2, (int)ctx->cfg.ring_stages));
  out->n_slots = n;
  out->bytes = (size_t)out->ring_off + (size_t)n * g.slot_bytes;
  return WISP_OK;
}

// A grid barrier of the fused kernel timed out in an earlier launch: report it once, put the device-side protocol state back.
int check_dev_err(wisp_ctx* ctx) {
  if (!ctx->host_err || !*reinterpret_cast<volatile int*>(ctx->host_err)) return WISP_OK;
  cudaDeviceSynchronize();
  *reinterpret_cast<volatile int*>(ctx->host_err) = 0;
  cudaMemset(ctx->zfix, 0, 2 * kZfixCopies * (size_t)kDecodeMaxTokens * ctx->cfg.n_experts * sizeof(long long));
  cudaMemset(ctx->dsync, 0, 4 * sizeof(unsigned));
  return fail(ctx, WISP_ECUDA, "fused decode kernel: a grid-wide barrier timed out; the outputs of that forward are invalid");
}

template <typename T, bool F8 = false>
int launch_fused(wisp_ctx* ctx, int lo, int hi, const void* x, int T_, void* out, bool residual, cudaStream_t st) {
  const auto& cfg = ctx->cfg;
  DecodeArgs pa{};
  pa.L = cfg.n_layers; pa.E = cfg.n_experts; pa.k = cfg.top_k; pa.d = cfg.d_model; pa.dff = cfg.d_ff; pa.T = T_; pa.C = ctx->C;
  pa.policy = cfg.policy; pa.wave_order = ctx->wave_order; pa.layer_lo = lo; pa.layer_hi = hi; pa.residual = residual ? 1 : 0;
  pa.pool = ctx->arena; pa.masters = reinterpret_cast<const char* const*>(ctx->d_masters); pa.blob_bytes = ctx->Me;
  pa.router_wt = ctx->router_wt; pa.router_bias = ctx->router_bias;
  pa.pi = ctx->pi; pa.pi_inv = ctx->pi_inv; pa.tau = ctx->tau; pa.freq = ctx->freq; pa.scal = ctx->scal;
  pa.last_pos = ctx->last_pos; pa.hist = ctx->hist;
  pa.logits = ctx->logits; pa.ids = ctx->ids; pa.topw = ctx->topw; pa.max_tokens = cfg.max_tokens;
  pa.partial = ctx->partial; pa.zfix = ctx->zfix; pa.sync = ctx->dsync;
  pa.x_in = x; pa.xbuf[0] = ctx->xbuf[0]; pa.xbuf[1] = ctx->xbuf[1]; pa.out = out;
  pa.err = ctx->dev_err;
  pa.trace = ctx->trace; pa.trace_ctr = ctx->trace_ctr; pa.trace_cap = ctx->trace_cap; pa.trace_on = ctx->trace_on;
  pa.track = ctx->track;
  pa.phase_ns = ctx->timing_level >= 2 ? ctx->phase_ns : nullptr;
  DecodeGeom g = ctx->dgeom[T_ <= 2 ? 0 : 1];
  DecodeSmem sm;
  int rc = decode_smem(ctx, g, T_, ctx->fused_smem, true, &sm);
  if (rc) return rc;
  CK(cudaMemsetAsync(ctx->dsync, 0, 4 * sizeof(unsigned), st));
  void* args[] = {&pa, &g, &sm.n_slots, &sm.xs_pitch, &sm.pre_off, &sm.ring_off};
  CK(cudaLaunchCooperativeKernel(T_ > 1 ? (const void*)decode_fused_kernel<T, F8, true> : (const void*)decode_fused_kernel<T, F8, false>, dim3(ctx->num_sms), dim3(kDecThreads), args, sm.bytes, st));
  ++ctx->launches;
  for (int l = lo; l < hi; ++l) ctx->last_T[l] = T_;
  ctx->last_layer = hi - 1;
  if (ctx->timing_level >= 2) ctx->fused_layers_timed += (u64)(hi - lo);
  return WISP_OK;
}

int launch_fused_any(wisp_ctx* ctx, int lo, int hi, const void* x, int T_, void* out, bool residual, cudaStream_t st) {
  if (ctx->f8) return launch_fused<__nv_bfloat16, true>(ctx, lo, hi, x, T_, out, residual, st);
  return ctx->cfg.dtype == WISP_F32 ? launch_fused<float>(ctx, lo, hi, x, T_, out, residual, st)
                                    : launch_fused<__nv_bfloat16>(ctx, lo, hi, x, T_, out, residual, st);
}

// Split form of one decode layer (MEMCPY / ZEROCOPY contexts, E > 256): logits, plan, per wave (fetch, ffn), combine -- the
// same device functions as the fused kernel, so both give the same bits.  x_next != nullptr: residual successor instead of y.
template <typename T, bool F8 = false>
int forward_layer_decode(wisp_ctx* ctx, int layer, const void* x, int T_, void* out, void* x_next, cudaStream_t st,
                         const char* slot_base = nullptr) {
  const auto& cfg = ctx->cfg;
  const int k = cfg.top_k, E = cfg.n_experts, d = cfg.d_model, L = cfg.n_layers;
  const int n_pairs = T_ * k, n_slices = T_ * (d / kSliceCols);
  const size_t off = (size_t)layer * cfg.max_tokens * k;
  const bool memcpy_path = cfg.fetch == WISP_FETCH_MEMCPY;
  const T* wrt = reinterpret_cast<const T*>(ctx->router_wt) + (size_t)layer * d * E;
  if (ctx->pf_n > 0 && ctx->pf_pending[layer]) {               // speculative copies into this layer's slots come first
    CK(cudaStreamWaitEvent(st, ctx->ev_copied[layer], 0));
    ctx->pf_pending[layer] = 0;
  }
  {
    Span sp(ctx, WISP_K_ROUTER, st);
    decode_logits_kernel<T><<<std::min(n_slices, 4 * ctx->num_sms), 256, 0, st>>>(reinterpret_cast<const T*>(x), wrt, ctx->zfix, T_, E, d);
  }
  {
    PlanArgs a;
    a.ids = nullptr; a.n_pairs = n_pairs; a.E = E; a.C = ctx->C; a.policy = cfg.policy; a.layer = layer;
    a.st = layer_state(ctx, layer); a.plan = ctx->plan; a.host_plan = memcpy_path ? ctx->host_plan : nullptr;
    a.trace = ctx->trace; a.trace_ctr = ctx->trace_ctr; a.trace_cap = ctx->trace_cap; a.trace_on = ctx->trace_on;
    a.wave_order = ctx->wave_order; a.track = ctx->track; a.build_pairs = 1;
    Span sp(ctx, WISP_K_RESIDENCY, st);
    const float* bias = ctx->router_bias + (size_t)layer * E;
    if (E <= 256) decode_plan_kernel<256><<<1, 256, 0, st>>>(a, ctx->zfix, bias, ctx->logits, ctx->ids + off, ctx->topw + off, T_, k);
    else decode_plan_kernel<kPlanThreads><<<1, kPlanThreads, 0, st>>>(a, ctx->zfix, bias, ctx->logits, ctx->ids + off, ctx->topw + off, T_, k);
  }
  CK(cudaGetLastError());
  if (ctx->pf_n > 0) {
    // f3: the predictor learns this layer's routing and prefetches for layer + 1 on the side stream while this layer computes
    PredictArgs pa{};
    pa.L = L; pa.E = E; pa.C = ctx->C; pa.policy = cfg.policy; pa.layer = layer; pa.window = ctx->pf_window; pa.n_prefetch = ctx->pf_n;
    for (int i = 0; i <= kMaxWindow; ++i) pa.gpow[i] = ctx->pf_gpow[i];
    pa.entry_expert = ctx->plan.entry_expert; pa.plan_hdr = ctx->plan.hdr;
    pa.A = ctx->pf_A; pa.row = ctx->pf_row; pa.rlist = ctx->pf_rlist; pa.rcount = ctx->pf_rcount;
    pa.st_next = layer_state(ctx, std::min(layer + 1, L - 1));
    pa.copy_list = ctx->pf_copy + (size_t)layer * (1 + 2 * kMaxPrefetch);
    pa.trace = ctx->trace; pa.trace_ctr = ctx->trace_ctr; pa.trace_cap = ctx->trace_cap; pa.trace_on = ctx->trace_on;
    {
      Span sp(ctx, WISP_K_OTHER, st);
      predict_prefetch_kernel<<<1, kPredictThreads, 0, st>>>(pa);
    }
    if (layer + 1 < L) {
      CK(cudaEventRecord(ctx->ev_pred[layer], st));
      CK(cudaStreamWaitEvent(ctx->pf_stream, ctx->ev_pred[layer], 0));
      prefetch_copy_kernel<<<32, 256, 0, ctx->pf_stream>>>(pa.copy_list, reinterpret_cast<const uint4*>(ctx->master[layer + 1]),
                                                         reinterpret_cast<uint4*>(ctx->arena), ctx->Me / 16, L, layer + 1);
      ++ctx->launches;
      CK(cudaEventRecord(ctx->ev_copied[layer + 1], ctx->pf_stream));
      ctx->pf_pending[layer + 1] = 1;
    }
    CK(cudaGetLastError());
  }
  int n_waves;
  if (memcpy_path) {
    CK(cudaEventRecord(ctx->ev_plan, st));
    CK(cudaEventSynchronize(ctx->ev_plan));      // the host must see the miss list
    n_waves = ctx->host_plan->n_waves;
  } else {
    n_waves = (std::min(E, n_pairs) + ctx->C - 1) / ctx->C;   // worst case; empty waves exit at once
  }
  const DecodeGeom g = ctx->dgeom[T_ <= 2 ? 0 : 1];
  DecodeSmem sm;
  int rc = decode_smem(ctx, g, T_, ctx->ffn_smem, false, &sm);
  if (rc) return rc;
  DecodeFfnArgs fa{};
  fa.layer_base = slot_base ? slot_base : ctx->arena + (size_t)layer * ctx->Me;
  fa.slot_stride = slot_base ? ctx->Me : (u64)L * ctx->Me;
  fa.blob_bytes = ctx->Me; fa.k = k; fa.partial = ctx->partial;
  fa.master = cfg.fetch == WISP_FETCH_FUSED ? static_cast<const char*>(ctx->master[layer]) : nullptr;
  fa.ticket = ctx->dsync + 1;
  for (int w = 0; w < n_waves; ++w) {
    if (cfg.fetch != WISP_FETCH_FUSED && cfg.fetch != WISP_FETCH_STATIC) {
      rc = fetch_wave(ctx, layer, w, memcpy_path, st);
      if (rc) return rc;
    }
    CK(cudaMemsetAsync(ctx->dsync + 1, 0, sizeof(unsigned), st));
    Span sp(ctx, WISP_K_FFN, st);
    decode_ffn_kernel<T, F8><<<ctx->num_sms, kDecThreads, sm.bytes, st>>>(fa, g, ctx->plan, w, ctx->C, E, T_, reinterpret_cast<const T*>(x),
                                                                     sm.n_slots, sm.xs_pitch, sm.ring_off);
  }
  {
    CombineArgs ca;
    ca.partial = ctx->partial; ca.n_chunks = g.n_chunks; ca.d = d; ca.k = k; ca.topw = ctx->topw + off; ca.pair_pos = ctx->plan.pair_pos;
    Span sp(ctx, WISP_K_COMBINE, st);
    decode_combine_kernel<T><<<std::min(n_slices, 4 * ctx->num_sms), 256, 0, st>>>(
        ca, x_next ? reinterpret_cast<const T*>(x) : nullptr, reinterpret_cast<T*>(x_next ? x_next : out), T_);
  }
  CK(cudaGetLastError());
  ctx->last_T[layer] = T_;
  ctx->last_layer = layer;
  return WISP_OK;
}

// ---- prefill path: grouped GEMM per wave (n_tokens > kDecodeMaxTokens) ----------------------------------------------
template <typename T, bool F8 = false>
int launch_prefill_wave(wisp_ctx* ctx, int layer, int wave, const void* x, int T_, cudaStream_t st) {
  const auto& cfg = ctx->cfg;
  const int d = cfg.d_model, dff = cfg.d_ff, k = cfg.top_k, L = cfg.n_layers;
  const T* pool = reinterpret_cast<const T*>(ctx->arena);
  if (ctx->mma_ok) {
    // tcgen05 grouped GEMM (bf16): xg was gathered once per forward (forward_layer_prefill); 4 / 6 ring stages of 48 / 32 KiB
    MmaArgs m{};
    m.plan = ctx->plan; m.wave = wave; m.C = ctx->C; m.L = L; m.layer = layer; m.d = d; m.dff = dff; m.k = k;
    m.act = reinterpret_cast<__nv_bfloat16*>(ctx->act_T); m.ystage = ctx->ystage;
    int* n_work = ctx->mma_work + 4 * (cfg.n_experts + cfg.max_tokens * k / kMmaNT + 1);
    {
      Span sp(ctx, WISP_K_OTHER, st);
      build_work_kernel<<<1, 32, 0, st>>>(ctx->plan, wave, ctx->C, ctx->mma_work, n_work);
    }
    {
      Span sp(ctx, WISP_K_PREFILL_GATE_UP, st);
      const int ns = 4;
      prefill_mma_kernel<0><<<ctx->num_sms, kMmaThreads, ns * 3 * kMmaTileBytes + 1024, st>>>(ctx->tm_gu, ctx->tm_xg, m, ctx->mma_work, n_work, ns);
    }
    {
      Span sp(ctx, WISP_K_PREFILL_DOWN, st);
      const int ns = 4;
      prefill_mma_kernel<1><<<ctx->num_sms, kMmaThreads, ns * 3 * kMmaTileBytes + 1024, st>>>(ctx->tm_dn, ctx->tm_act, m, ctx->mma_work, n_work, ns);
    }
  } else {
    const int ptiles = (T_ + kPfTile - 1) / kPfTile;   // an expert can receive at most T pairs
    dim3 g0(dff / kPfTile, ptiles, ctx->C), g1(d / kPfTile, ptiles, ctx->C);
    {
      Span sp(ctx, WISP_K_PREFILL_GATE_UP, st);
      prefill_ffn_kernel<T, 0, F8><<<g0, 256, 0, st>>>(ctx->plan, wave, ctx->C, pool, F8 ? ctx->Me : ctx->blob_elems, L, layer,
                                                       reinterpret_cast<const T*>(x), reinterpret_cast<T*>(ctx->act_T),
                                                       ctx->ystage, d, dff, k, ctx->s13_off, ctx->s2_off);
    }
    {
      Span sp(ctx, WISP_K_PREFILL_DOWN, st);
      prefill_ffn_kernel<T, 1, F8><<<g1, 256, 0, st>>>(ctx->plan, wave, ctx->C, pool, F8 ? ctx->Me : ctx->blob_elems, L, layer,
                                                       reinterpret_cast<const T*>(x), reinterpret_cast<T*>(ctx->act_T),
                                                       ctx->ystage, d, dff, k, ctx->s13_off, ctx->s2_off);
    }
  }
  CK(cudaGetLastError());
  return WISP_OK;
}

// Tensor maps of the tcgen05 prefill path.  Weights: 4-D views of the arena in the tiled in-slot layout (common.cuh),
// (64 elements of a core matrix, core column, core row, blob = slot*L + layer), no swizzle; tokens / activations: 2-D
// K-major views of xg and act with the 128-byte swizzle; router rows: 3-D row-major view with the 128-byte swizzle.
bool setup_mma_path(wisp_ctx* ctx) {
  const auto& cfg = ctx->cfg;
  if (cfg.dtype != WISP_BF16 || cfg.max_tokens <= kDecodeMaxTokens) return false;
  void* sym = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) != cudaSuccess || !sym) return false;
  EncodeTiledFn fn = reinterpret_cast<EncodeTiledFn>(sym);
  ctx->encode_fn = sym;
  const cuuint64_t d = cfg.d_model, dff = cfg.d_ff, n_blobs = ctx->budget / ctx->Me, rows = (cuuint64_t)cfg.max_tokens * cfg.top_k;
  if (n_blobs < 1) return false;
  const cuuint32_t box3[3] = {kMmaBK, kMmaM, 1}, box2[2] = {kMmaBK, kMmaNT};
  {
    // gate then up: core (r/8, k/8) at ((r/8)*(d/8) + k/8) * 128 B; a tile = 16 row groups x 8 K cores
    const cuuint64_t dims[4] = {64, d / 8, 2 * dff / 8, n_blobs}, str[3] = {128, d * 16, ctx->Me};
    const cuuint32_t box[4] = {64, kMmaBK / 8, kMmaM / 8, 1};
    if (!make_tmap(fn, &ctx->tm_gu, ctx->arena, 4, dims, str, box, false)) return false;
  }
  {
    // down: core (j/8, i/8) at ((i/8)*(d/8) + j/8) * 128 B; a tile = 8 act-column blocks x 16 output groups
    const cuuint64_t dims[4] = {64, d / 8, dff / 8, n_blobs}, str[3] = {128, d * 16, ctx->Me};
    const cuuint32_t box[4] = {64, kMmaM / 8, kMmaBK / 8, 1};
    if (!make_tmap(fn, &ctx->tm_dn, ctx->arena + 2 * d * dff * 2, 4, dims, str, box, false)) return false;
  }
  if (cudaMalloc(&ctx->xg, rows * d * 2) != cudaSuccess) return false;
  if (cudaMalloc(&ctx->mma_work, (4 * (size_t)(cfg.n_experts + cfg.max_tokens * cfg.top_k / kMmaNT + 1) + 4) * sizeof(int)) != cudaSuccess) return false;
  {
    const cuuint64_t dims[2] = {d, rows}, str[1] = {d * 2};
    if (!make_tmap(fn, &ctx->tm_xg, ctx->xg, 2, dims, str, box2, true)) return false;
  }
  {
    const cuuint64_t dims[2] = {dff, rows}, str[1] = {dff * 2};
    if (!make_tmap(fn, &ctx->tm_act, ctx->act_T, 2, dims, str, box2, true)) return false;
  }
  if (cfg.n_experts % kMmaM == 0) {   // router weights [L][E][d] as (K, expert row, layer)
    const cuuint64_t dims[3] = {d, (cuuint64_t)cfg.n_experts, (cuuint64_t)cfg.n_layers}, str[2] = {d * 2, (cuuint64_t)cfg.n_experts * d * 2};
    if (!make_tmap(fn, &ctx->tm_rw, ctx->router_w, 3, dims, str, box3, true)) return false;
  }
  for (int mode = 0; mode < 3; ++mode) {
    const void* k = mode == 0 ? (const void*)prefill_mma_kernel<0> : mode == 1 ? (const void*)prefill_mma_kernel<1> : (const void*)prefill_mma_kernel<2>;
    if (cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024) != cudaSuccess) return false;
  }
  return true;
}

// One prefill MoE layer: router -> residency -> per wave (fetch, grouped GEMMs into ystage [T,k,d]) -> ordered combine (a5).
template <typename T, bool F8 = false>
int forward_layer_prefill(wisp_ctx* ctx, int layer, const void* x, int T_, void* out, void* x_next, cudaStream_t st) {
  const auto& cfg = ctx->cfg;
  const int k = cfg.top_k, E = cfg.n_experts;
  const int n_pairs = T_ * k;
  int rc = launch_router<T>(ctx, layer, x, T_, st);
  if (rc) return rc;
  const size_t off = (size_t)layer * cfg.max_tokens * k;
  const bool memcpy_path = cfg.fetch == WISP_FETCH_MEMCPY;
  rc = launch_plan(ctx, layer, ctx->ids + off, n_pairs, memcpy_path, st);
  if (rc) return rc;
  int n_waves;
  if (memcpy_path) {
    CK(cudaEventRecord(ctx->ev_plan, st));
    CK(cudaEventSynchronize(ctx->ev_plan));      // the host must see the miss list
    n_waves = ctx->host_plan->n_waves;
  } else {
    n_waves = (std::min(E, n_pairs) + ctx->C - 1) / ctx->C;   // worst case; empty waves exit at once
  }
  if (ctx->mma_ok) {                               // B operand of GEMM 1: token rows in sorted-pair order
    Span sp(ctx, WISP_K_OTHER, st);
    gather_tokens_kernel<<<std::min((n_pairs + 7) / 8, 8 * ctx->num_sms), 256, 0, st>>>(ctx->plan.pair_list, n_pairs, k, cfg.d_model * 2 / 16,
                                                                             reinterpret_cast<const uint4*>(x), reinterpret_cast<uint4*>(ctx->xg));
  }
  for (int w = 0; w < n_waves; ++w) {
    rc = fetch_wave(ctx, layer, w, memcpy_path, st);   // prefill under FUSED uses the zero-copy kernel
    if (rc) return rc;
    rc = launch_prefill_wave<T, F8>(ctx, layer, w, x, T_, st);
    if (rc) return rc;
  }
  const size_t n = (size_t)T_ * cfg.d_model;
  {
    Span sp(ctx, WISP_K_COMBINE, st);
    combine_kernel<T><<<(unsigned)((n / 4 + 255) / 256), 256, 0, st>>>(ctx->ystage, ctx->topw + off, reinterpret_cast<T*>(out),
                                                                   x_next ? reinterpret_cast<const T*>(x) : nullptr,
                                                                   reinterpret_cast<T*>(x_next), T_, cfg.d_model, k);
  }
  CK(cudaGetLastError());
  ctx->last_T[layer] = T_;
  ctx->last_layer = layer;
  return WISP_OK;
}

int forward_layer_any(wisp_ctx* ctx, int layer, const void* x, int T_, void* out, void* x_next, cudaStream_t st) {
  const bool f32 = ctx->cfg.dtype == WISP_F32;
  if (ctx->f8)
    return T_ <= kDecodeMaxTokens ? forward_layer_decode<__nv_bfloat16, true>(ctx, layer, x, T_, out, x_next, st)
                                  : forward_layer_prefill<__nv_bfloat16, true>(ctx, layer, x, T_, out, x_next, st);
  if (T_ <= kDecodeMaxTokens)
    return f32 ? forward_layer_decode<float>(ctx, layer, x, T_, out, x_next, st)
               : forward_layer_decode<__nv_bfloat16>(ctx, layer, x, T_, out, x_next, st);
  return f32 ? forward_layer_prefill<float>(ctx, layer, x, T_, out, x_next, st)
             : forward_layer_prefill<__nv_bfloat16>(ctx, layer, x, T_, out, x_next, st);
}

// ---- static layer-offload arm (comparison) --------------------------------------------------------
// Copy of all E experts of `layer` into bounce buffer `layer & 1` on the copy stream, after the compute that last used the
// buffer.  No residency cache: a streamed layer is copied again on every forward.
int static_issue_copy(wisp_ctx* ctx, int layer) {
  const int b = layer & 1;
  const u64 layer_bytes = (u64)ctx->cfg.n_experts * ctx->Me;
  if (ctx->buf_used[b]) CK(cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_buf_free[b], 0));
  CK(cudaMemcpyAsync(ctx->bounce[b], ctx->master[layer], layer_bytes, cudaMemcpyHostToDevice, ctx->copy_stream));
  CK(cudaEventRecord(ctx->ev_buf_ready[b], ctx->copy_stream));
  ctx->static_streamed += layer_bytes;
  return WISP_OK;
}

// One layer of the static arm on stream st.  copy_issued: the caller already queued this layer's copy (stack helper, which
// streams layer l+1 while layer l computes).
int forward_layer_static(wisp_ctx* ctx, int layer, const void* x, int T_, void* out, void* x_next, cudaStream_t st, bool copy_issued) {
  const bool resident = layer < ctx->static_pinned;
  const int b = layer & 1;
  const char* base = resident ? ctx->arena + (u64)layer * ctx->cfg.n_experts * ctx->Me : ctx->bounce[b];
  if (!resident) {
    if (!copy_issued) {
      int rc = static_issue_copy(ctx, layer);
      if (rc) return rc;
    }
    CK(cudaStreamWaitEvent(st, ctx->ev_buf_ready[b], 0));
  }
  int rc = ctx->f8 ? forward_layer_decode<__nv_bfloat16, true>(ctx, layer, x, T_, out, x_next, st, base)
           : ctx->cfg.dtype == WISP_F32 ? forward_layer_decode<float>(ctx, layer, x, T_, out, x_next, st, base)
                                        : forward_layer_decode<__nv_bfloat16>(ctx, layer, x, T_, out, x_next, st, base);
  if (rc) return rc;
  if (!resident) {
    CK(cudaEventRecord(ctx->ev_buf_free[b], st));
    ctx->buf_used[b] = true;
  }
  return WISP_OK;
}

int check_forward_args(wisp_ctx* ctx, int layer_lo, int layer_hi, const void* hidden, int n_tokens, void* out) {
  if (!ctx) return WISP_EINVAL;
  if (n_tokens < 0 || n_tokens > ctx->cfg.max_tokens) return fail(ctx, WISP_EINVAL, "n_tokens out of range");
  if (n_tokens > 0 && (!hidden || !out)) return fail(ctx, WISP_EINVAL, "null hidden/out");
  for (int l = layer_lo; l < layer_hi; ++l) {
    if (l < 0 || l >= ctx->cfg.n_layers) return fail(ctx, WISP_EINVAL, "layer out of range");
    if (!ctx->registered[l]) return fail(ctx, WISP_ESTATE, "layer not registered");
  }
  return WISP_OK;
}

template <typename F>
int occupancy_grid(wisp_ctx* ctx, F kernel, int threads, int cap_per_sm) {
  int nb = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kernel, threads, 0) != cudaSuccess || nb < 1) nb = 1;
  return ctx->num_sms * std::min(nb, cap_per_sm);
}


// Re-tile the caller's canonical blobs ([gate | up | down], row-major out x in) into the in-slot layout of common.cuh:
// 8-row x 16-byte core matrices, gate/up cores ordered (row group, K), down cores ordered (act-column block, output group).
// Pure byte movement in 16-byte pieces, spread over host threads (a layer is 1-3 GiB).
// fp8 blobs: the codes of gate / up tile the same way (16 codes per 16-byte row of a core); down uses 8-output x 8-column cores of
// 64 bytes (one decode work unit owns 8 act columns); the scales follow: S13 as given, S2 transposed to [d_ff / 128][d / 128].
void retile_layer(const char* src, char* dst, size_t E, size_t d, size_t dff, size_t elem, bool f8) {
  const size_t kc = 16 / elem, mat = d * dff * elem;
  const size_t n13 = f8 ? (2 * dff / 128) * (d / 128) : 0, n2 = f8 ? (d / 128) * (dff / 128) : 0;
  const size_t Me = 3 * mat + 4 * (n13 + n2);
  const size_t gu_items = E * 2 * (dff / 8);                 // (expert, gate|up, row group)
  const size_t ib_per = dff / kc, line_ib = std::max<size_t>(1, 64 / 16);   // down: 4 act-column blocks share a 64-byte line
  const size_t dn_items = E * ((ib_per + line_ib - 1) / line_ib);
  const size_t total = gu_items + dn_items;
  const unsigned hw = std::thread::hardware_concurrency();
  const size_t nthr = std::min<size_t>(32, std::max<size_t>(4, hw ? hw : 8));
  auto work = [=](size_t lo, size_t hi) {
    for (size_t it = lo; it < hi; ++it) {
      if (it < gu_items) {
        const size_t e = it / (2 * (dff / 8)), rem = it % (2 * (dff / 8)), m = rem / (dff / 8), rg = rem % (dff / 8);
        const char* s0 = src + e * Me + m * mat + rg * 8 * d * elem;
        char* o = dst + e * Me + m * mat + rg * 8 * d * elem;
        for (size_t kb = 0; kb < d / kc; ++kb)
          for (size_t r = 0; r < 8; ++r) std::memcpy(o + (kb * 8 + r) * 16, s0 + r * d * elem + kb * 16, 16);
      } else {
        const size_t q = it - gu_items, groups = (ib_per + line_ib - 1) / line_ib, e = q / groups, ib0 = (q % groups) * line_ib;
        const size_t nib = std::min(line_ib, ib_per - ib0);
        const char* s0 = src + e * Me + 2 * mat;             // down [d][dff]
        char* o = dst + e * Me + 2 * mat;
        if (f8) {
          for (size_t j = 0; j < d; ++j)
            for (size_t b = 0; b < 2 * nib; ++b)               // 8-column blocks
              std::memcpy(o + (((ib0 * 2 + b) * (d / 8) + j / 8) * 8 + (j & 7)) * 8, s0 + j * dff + (ib0 * 2 + b) * 8, 8);
          if (ib0 == 0) {                                      // this expert's scales (once)
            const float* sc = reinterpret_cast<const float*>(src + e * Me + 3 * mat);
            float* so = reinterpret_cast<float*>(dst + e * Me + 3 * mat);
            std::memcpy(so, sc, 4 * n13);
            for (size_t jb = 0; jb < d / 128; ++jb)
              for (size_t cb = 0; cb < dff / 128; ++cb) so[n13 + cb * (d / 128) + jb] = sc[n13 + jb * (dff / 128) + cb];
          }
          continue;
        }
        for (size_t j = 0; j < d; ++j)
          for (size_t b = 0; b < nib; ++b)
            std::memcpy(o + (((ib0 + b) * (d / 8) + j / 8) * 8 + (j & 7)) * 16, s0 + (j * dff + (ib0 + b) * kc) * elem, 16);
      }
    }
  };
  std::vector<std::thread> th;
  const size_t per = (total + nthr - 1) / nthr;
  for (size_t i = 0; i < nthr; ++i) {
    const size_t lo = i * per, hi = std::min(total, lo + per);
    if (lo >= hi) break;
    th.emplace_back(work, lo, hi);
  }
  for (auto& t : th) t.join();
}

}  // namespace

extern "C" {

const char* wisp_version(void) { return kVersion; }


const char* wisp_last_error(wisp_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int wisp_create(uint64_t budget_bytes, const wisp_config* cfg, wisp_ctx** out) {
  if (!cfg || !out) return WISP_EINVAL;
  *out = nullptr;
  if (cfg->n_layers < 1 || cfg->n_experts < 1 || cfg->n_experts > kMaxExperts || cfg->top_k < 1 ||
      cfg->top_k > kMaxTopK || cfg->top_k > cfg->n_experts || cfg->d_model < 256 || cfg->d_model % 256 ||
      cfg->d_ff < 256 || cfg->d_ff % 256 || cfg->max_tokens < 1 ||
      (cfg->dtype != WISP_F32 && cfg->dtype != WISP_BF16 && cfg->dtype != WISP_FP8_E4M3) ||
      (cfg->dtype == WISP_FP8_E4M3 && cfg->d_model % 1024) || (cfg->policy != WISP_LRU && cfg->policy != WISP_LFU) ||
      (cfg->fetch != WISP_FETCH_MEMCPY && cfg->fetch != WISP_FETCH_ZEROCOPY && cfg->fetch != WISP_FETCH_FUSED &&
       cfg->fetch != WISP_FETCH_STATIC) ||
      cfg->ring_stages < 0 || cfg->ring_stages > kDecMaxSlots || cfg->unit_rows < 0 || cfg->unit_rows % 8 ||
      (cfg->unit_rows > 0 && (cfg->d_ff % cfg->unit_rows || (cfg->d_ff / cfg->unit_rows) % 8)))
    return WISP_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return WISP_ECUDA;   // no CPU fallback
  wisp_ctx* ctx = new wisp_ctx();
  ctx->cfg = *cfg;
  ctx->budget = budget_bytes;
  ctx->elem = cfg->dtype == WISP_F32 ? 4 : 2;
  ctx->f8 = cfg->dtype == WISP_FP8_E4M3;
  ctx->welem = ctx->f8 ? 1 : ctx->elem;
  ctx->blob_elems = 3 * (size_t)cfg->d_model * cfg->d_ff;
  ctx->Me = ctx->blob_elems * ctx->welem;
  if (ctx->f8) {                                   // + the fp32 block scales S13 and S2 (one per 128 x 128 block)
    ctx->s13_off = ctx->Me;
    ctx->s2_off = ctx->s13_off + 4 * (size_t)(2 * cfg->d_ff / 128) * (cfg->d_model / 128);
    ctx->Me = ctx->s2_off + 4 * (size_t)(cfg->d_model / 128) * (cfg->d_ff / 128);
  }
  ctx->a_bytes = ctx->Me * cfg->n_layers;
  const u64 b = cfg->kv_block_bytes;
  const u64 kv0 = b ? cfg->kv_floor_blocks * b : 0;
  if (kv0 > budget_bytes || (budget_bytes - kv0) / ctx->a_bytes < 1) {
    delete ctx;
    return WISP_EBUDGET;
  }
  ctx->C = (int)std::min<u64>(cfg->n_experts, (budget_bytes - kv0) / ctx->a_bytes);
  if (cfg->fetch == WISP_FETCH_STATIC) {
    // whole layers: floor(B / (E*M_e)) - 2 resident, 2 as bounce buffers; every expert of a layer is "resident" while it runs
    const u64 layer_bytes = (u64)cfg->n_experts * ctx->Me;
    if (kv0 != 0 || budget_bytes / layer_bytes < 2 || cfg->max_tokens > kDecodeMaxTokens) {
      delete ctx;
      return cfg->max_tokens > kDecodeMaxTokens ? WISP_EINVAL : WISP_EBUDGET;
    }
    ctx->static_pinned = (int)std::min<u64>(cfg->n_layers, budget_bytes / layer_bytes - 2);
    ctx->C = cfg->n_experts;
  }
  ctx->kappa = b ? (budget_bytes - (u64)ctx->C * ctx->a_bytes) / b : 0;
  const int L = cfg->n_layers, E = cfg->n_experts, k = cfg->top_k, d = cfg->d_model, dff = cfg->d_ff;
  const size_t maxT = cfg->max_tokens;
  ctx->master.assign(L, nullptr);
  ctx->registered.assign(L, 0);
  ctx->last_T.assign(L, 0);
  ctx->host_hist.assign(E + 2, 0.0);
  ctx->trace_cap = cfg->trace_capacity ? cfg->trace_capacity : (1ull << 20);
  cudaDeviceProp prop;
  int dev = 0;
  auto bail = [&](int code, const char* what, cudaError_t e) {
    std::fprintf(stderr, "wisp_create: %s: %s\n", what, cudaGetErrorString(e));
    wisp_destroy(ctx);
    return code;
  };
#define CKC(call)                                                                                            \
  do {                                                                                                       \
    cudaError_t e_ = (call);                                                                                 \
    if (e_ != cudaSuccess) return bail(e_ == cudaErrorMemoryAllocation ? WISP_ENOMEM : WISP_ECUDA, #call, e_); \
  } while (0)
  CKC(cudaGetDevice(&dev));
  CKC(cudaGetDeviceProperties(&prop, dev));
  ctx->num_sms = prop.multiProcessorCount;
  CKC(cudaMalloc(&ctx->arena, budget_bytes));
  CKC(cudaMalloc(&ctx->router_w, (size_t)L * E * d * ctx->elem));
  CKC(cudaMalloc(&ctx->router_wt, (size_t)L * E * d * ctx->elem));
  CKC(cudaMalloc(&ctx->router_bias, (size_t)L * E * sizeof(float)));
  CKC(cudaMalloc(&ctx->pi, (size_t)L * E * sizeof(int)));
  CKC(cudaMalloc(&ctx->pi_inv, (size_t)L * E * sizeof(int)));
  CKC(cudaMalloc(&ctx->tau, (size_t)L * E * sizeof(u64)));
  CKC(cudaMalloc(&ctx->freq, (size_t)L * E * sizeof(u64)));
  CKC(cudaMalloc(&ctx->scal, (size_t)L * 8 * sizeof(u64)));
  CKC(cudaMalloc(&ctx->last_pos, (size_t)L * E * sizeof(u64)));
  CKC(cudaMalloc(&ctx->hist, (size_t)L * (E + 2) * sizeof(u64)));
  CKC(cudaMemset(ctx->pi, 0xff, (size_t)L * E * sizeof(int)));
  CKC(cudaMemset(ctx->pi_inv, 0xff, (size_t)L * E * sizeof(int)));
  CKC(cudaMemset(ctx->tau, 0, (size_t)L * E * sizeof(u64)));
  CKC(cudaMemset(ctx->freq, 0, (size_t)L * E * sizeof(u64)));
  CKC(cudaMemset(ctx->scal, 0, (size_t)L * 8 * sizeof(u64)));
  CKC(cudaMemset(ctx->last_pos, 0, (size_t)L * E * sizeof(u64)));
  CKC(cudaMemset(ctx->hist, 0, (size_t)L * (E + 2) * sizeof(u64)));
  CKC(cudaMalloc(&ctx->logits, maxT * E * sizeof(float)));
  CKC(cudaMalloc(&ctx->ids, (size_t)L * maxT * k * sizeof(int)));
  CKC(cudaMemset(ctx->ids, 0, (size_t)L * maxT * k * sizeof(int)));
  CKC(cudaMalloc(&ctx->topw, (size_t)L * maxT * k * sizeof(float)));
  {
    const size_t n_int = 4 + 3 * (size_t)E + E + (E + 1) + 2 * maxT * k + E;
    CKC(cudaMalloc(&ctx->plan_mem, n_int * sizeof(int)));
    CKC(cudaMemset(ctx->plan_mem, 0, n_int * sizeof(int)));
    int* p = ctx->plan_mem;
    ctx->plan.hdr = p; p += 4;
    ctx->plan.entry_expert = p; p += E;
    ctx->plan.entry_slot = p; p += E;
    ctx->plan.entry_miss = p; p += E;
    ctx->plan.exp_count = p; p += E;
    ctx->plan.exp_offset = p; p += E + 1;
    ctx->plan.pair_list = p; p += maxT * k;
    ctx->plan.pair_pos = p; p += maxT * k;
    ctx->plan.unit_entry = p;
  }
  CKC(cudaHostAlloc(&ctx->host_plan, sizeof(HostPlan), cudaHostAllocMapped));
  std::memset(ctx->host_plan, 0, sizeof(HostPlan));
  CKC(cudaMalloc(&ctx->act_T, maxT * k * dff * ctx->elem));
  CKC(cudaMalloc(&ctx->ystage, maxT * k * d * sizeof(float)));
  CKC(cudaMalloc(&ctx->xbuf[0], maxT * d * ctx->elem));
  CKC(cudaMalloc(&ctx->xbuf[1], maxT * d * ctx->elem));
  CKC(cudaMalloc(&ctx->ybuf, maxT * d * ctx->elem));
  CKC(cudaMalloc(&ctx->moves, (2 * (size_t)E + 1) * sizeof(int)));
  CKC(cudaMalloc(&ctx->bad_slots, (size_t)E * sizeof(int)));
  CKC(cudaMalloc(&ctx->trace, ctx->trace_cap * sizeof(wisp_trace_event)));
  CKC(cudaMalloc(&ctx->trace_ctr, 2 * sizeof(u64)));
  CKC(cudaMemset(ctx->trace_ctr, 0, 2 * sizeof(u64)));
  CKC(cudaMalloc(&ctx->d_masters, (size_t)L * sizeof(char*)));
  CKC(cudaMemset(ctx->d_masters, 0, (size_t)L * sizeof(char*)));
  CKC(cudaMalloc(&ctx->dsync, 4 * sizeof(unsigned)));
  CKC(cudaMemset(ctx->dsync, 0, 4 * sizeof(unsigned)));
  CKC(cudaMalloc(&ctx->zfix, 2 * kZfixCopies * (size_t)kDecodeMaxTokens * E * sizeof(long long)));
  CKC(cudaMemset(ctx->zfix, 0, 2 * kZfixCopies * (size_t)kDecodeMaxTokens * E * sizeof(long long)));
  CKC(cudaHostAlloc(&ctx->host_err, sizeof(int), cudaHostAllocMapped));
  *ctx->host_err = 0;
  CKC(cudaHostGetDevicePointer(reinterpret_cast<void**>(&ctx->dev_err), ctx->host_err, 0));
  CKC(cudaMalloc(&ctx->phase_ns, (kDecPhases + 2) * sizeof(u64)));
  CKC(cudaMemset(ctx->phase_ns, 0, (kDecPhases + 2) * sizeof(u64)));
  {
    // Work-unit size of the decode FFN: 16 act rows (two sub-blocks of 8: 192 KiB of bf16 weights at the Qwen3 shape) -- the two
    // sub-blocks' down parts feed one MMA pass with all 16 k slots used, and a pair has half as many chunk partials to combine.
    // fp32 models (config 1, parity only) always use 8.
    const int r0 = cfg->unit_rows > 0 && cfg->dtype != WISP_F32 ? cfg->unit_rows : cfg->dtype == WISP_F32 ? 8 : 16;
    const int r1 = cfg->dtype == WISP_F32 ? 8 : cfg->unit_rows > 0 ? cfg->unit_rows : 16;
    ctx->dgeom[0] = make_decode_geom(d, dff, ctx->welem, r0, ctx->f8);
    ctx->dgeom[1] = make_decode_geom(d, dff, ctx->welem, r1, ctx->f8);
    const size_t t_dec = std::min<size_t>(maxT, kDecodeMaxTokens);
    const size_t pairs0 = std::min<size_t>(t_dec, 2) * k, pairs1 = t_dec * k;
    const size_t n_part = std::max(pairs0 * ctx->dgeom[0].n_chunks, pairs1 * ctx->dgeom[1].n_chunks) * d;
    CKC(cudaMalloc(&ctx->partial, n_part * sizeof(float)));
    cudaFuncAttributes fa;
    const void* kf = ctx->f8 ? (const void*)decode_fused_kernel<__nv_bfloat16, true, false>
                     : cfg->dtype == WISP_F32 ? (const void*)decode_fused_kernel<float, false, false> : (const void*)decode_fused_kernel<__nv_bfloat16, false, false>;
    const void* kf2 = ctx->f8 ? (const void*)decode_fused_kernel<__nv_bfloat16, true, true>
                      : cfg->dtype == WISP_F32 ? (const void*)decode_fused_kernel<float, false, true> : (const void*)decode_fused_kernel<__nv_bfloat16, false, true>;
    const void* kn = ctx->f8 ? (const void*)decode_ffn_kernel<__nv_bfloat16, true>
                     : cfg->dtype == WISP_F32 ? (const void*)decode_ffn_kernel<float, false> : (const void*)decode_ffn_kernel<__nv_bfloat16, false>;
    CKC(cudaFuncGetAttributes(&fa, kf));
    ctx->fused_smem = (227u << 10) - fa.sharedSizeBytes;
    CKC(cudaFuncSetAttribute(kf, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ctx->fused_smem));
    CKC(cudaFuncSetAttribute(kf2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ctx->fused_smem));
    CKC(cudaFuncGetAttributes(&fa, kn));
    ctx->ffn_smem = (227u << 10) - fa.sharedSizeBytes;
    CKC(cudaFuncSetAttribute(kn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ctx->ffn_smem));
  }
  if (ctx->is_static()) {
    // pi = pi^-1 = identity: slot e of a layer's region holds expert e
    std::vector<int> ident((size_t)L * E);
    for (size_t i = 0; i < ident.size(); ++i) ident[i] = (int)(i % E);
    CKC(cudaMemcpy(ctx->pi, ident.data(), ident.size() * sizeof(int), cudaMemcpyHostToDevice));
    CKC(cudaMemcpy(ctx->pi_inv, ident.data(), ident.size() * sizeof(int), cudaMemcpyHostToDevice));
    const u64 layer_bytes = (u64)E * ctx->Me;
    for (int b = 0; b < 2; ++b) {
      ctx->bounce[b] = ctx->arena + ((u64)ctx->static_pinned + b) * layer_bytes;
      CKC(cudaEventCreateWithFlags(&ctx->ev_buf_free[b], cudaEventDisableTiming));
      CKC(cudaEventCreateWithFlags(&ctx->ev_buf_ready[b], cudaEventDisableTiming));
    }
  }
  CKC(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
  CKC(cudaEventCreateWithFlags(&ctx->ev_plan, cudaEventDisableTiming));
  CKC(cudaEventCreateWithFlags(&ctx->ev_compute, cudaEventDisableTiming));
  CKC(cudaEventCreateWithFlags(&ctx->ev_copy, cudaEventDisableTiming));
#undef CKC
  ctx->grid_fetch = ctx->num_sms * 2;
  ctx->mma_ok = setup_mma_path(ctx);
  if (cfg->dtype == WISP_BF16 && cfg->max_tokens > kDecodeMaxTokens && !ctx->mma_ok) {
    std::fprintf(stderr, "wisp_create: tcgen05 prefill path unavailable (tensor map setup failed)\n");
    wisp_destroy(ctx);
    return WISP_ECUDA;
  }
  *out = ctx;
  return WISP_OK;
}

int wisp_destroy(wisp_ctx* ctx) {
  if (!ctx) return WISP_EINVAL;
  cudaDeviceSynchronize();
  drop_graphs(ctx);
  for (void* m : ctx->master)
    if (m) cudaFreeHost(m);
  void* dev_ptrs[] = {ctx->arena,    ctx->router_w, ctx->router_bias, ctx->pi,      ctx->pi_inv,  ctx->tau,
                      ctx->freq,     ctx->scal,     ctx->last_pos,    ctx->hist,    ctx->logits,  ctx->ids,
                      ctx->topw,     ctx->plan_mem, ctx->router_wt,   ctx->act_T,   ctx->ystage,  ctx->xbuf[0],
                      ctx->xbuf[1],  ctx->ybuf,     ctx->dbg_ids,     ctx->moves,   ctx->bad_slots, ctx->trace,
                      ctx->trace_ctr, ctx->d_masters, ctx->dsync, ctx->zfix, ctx->partial, ctx->phase_ns, ctx->xg, ctx->mma_work};
  for (void* p : dev_ptrs)
    if (p) cudaFree(p);
  if (ctx->host_plan) cudaFreeHost(ctx->host_plan);
  if (ctx->host_err) cudaFreeHost(ctx->host_err);
  for (void* p : {(void*)ctx->pf_A, (void*)ctx->pf_row, (void*)ctx->pf_rlist, (void*)ctx->pf_rcount, (void*)ctx->pf_copy})
    if (p) cudaFree(p);
  if (ctx->pf_stream) cudaStreamDestroy(ctx->pf_stream);
  for (cudaEvent_t e : ctx->ev_pred) cudaEventDestroy(e);
  for (cudaEvent_t e : ctx->ev_copied) cudaEventDestroy(e);
  if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
  for (cudaEvent_t e : {ctx->ev_plan, ctx->ev_compute, ctx->ev_copy, ctx->ev_buf_free[0], ctx->ev_buf_free[1], ctx->ev_buf_ready[0],
                        ctx->ev_buf_ready[1]})
    if (e) cudaEventDestroy(e);
  for (auto& p : ctx->timing_pool) {
    cudaEventDestroy(p.a);
    cudaEventDestroy(p.b);
  }
  delete ctx;
  return WISP_OK;
}

int wisp_register_host_experts(wisp_ctx* ctx, int32_t layer, const void* experts, const void* router_w,
                               const float* router_bias) {
  if (!ctx || !experts || !router_w) return fail(ctx, WISP_EINVAL, "null argument");
  if (layer < 0 || layer >= ctx->cfg.n_layers) return fail(ctx, WISP_EINVAL, "layer out of range");
  if (ctx->registered[layer]) return fail(ctx, WISP_ESTATE, "layer already registered");
  const size_t E = ctx->cfg.n_experts, d = ctx->cfg.d_model;
  void* m = nullptr;
  CK(cudaHostAlloc(&m, E * ctx->Me, cudaHostAllocMapped | cudaHostAllocPortable));
  retile_layer(static_cast<const char*>(experts), static_cast<char*>(m), E, d, ctx->cfg.d_ff, ctx->welem, ctx->f8);
  ctx->master[layer] = m;
  CK(cudaMemcpy(ctx->d_masters + layer, &m, sizeof(char*), cudaMemcpyHostToDevice));
  CK(cudaMemcpy(ctx->router_w + (size_t)layer * E * d * ctx->elem, router_w, E * d * ctx->elem, cudaMemcpyHostToDevice));
  {  // transposed copy [d][E] for the decode path's 16-column logit slices
    std::vector<char> wt(E * d * ctx->elem);
    const char* w = static_cast<const char*>(router_w);
    for (size_t e = 0; e < E; ++e)
      for (size_t j = 0; j < d; ++j) std::memcpy(wt.data() + (j * E + e) * ctx->elem, w + (e * d + j) * ctx->elem, ctx->elem);
    CK(cudaMemcpy(ctx->router_wt + (size_t)layer * E * d * ctx->elem, wt.data(), wt.size(), cudaMemcpyHostToDevice));
  }
  if (router_bias) CK(cudaMemcpy(ctx->router_bias + (size_t)layer * E, router_bias, E * sizeof(float), cudaMemcpyHostToDevice));
  else CK(cudaMemset(ctx->router_bias + (size_t)layer * E, 0, E * sizeof(float)));
  if (ctx->is_static() && layer < ctx->static_pinned)
    CK(cudaMemcpy(ctx->arena + (u64)layer * E * ctx->Me, m, E * ctx->Me, cudaMemcpyHostToDevice));
  ctx->registered[layer] = 1;
  return WISP_OK;
}

int wisp_moe_forward(wisp_ctx* ctx, int32_t layer, const void* hidden, int32_t n_tokens, void* out, void* cuda_stream) {
  int rc = check_forward_args(ctx, layer, layer + 1, hidden, n_tokens, out);
  if (rc) return rc;
  if (n_tokens == 0) return WISP_OK;
  if ((rc = check_dev_err(ctx))) return rc;
  if (ctx->is_static()) return forward_layer_static(ctx, layer, hidden, n_tokens, out, nullptr, static_cast<cudaStream_t>(cuda_stream), false);
  if (ctx->use_fused(n_tokens))
    return launch_fused_any(ctx, layer, layer + 1, hidden, n_tokens, out, false, static_cast<cudaStream_t>(cuda_stream));
  return forward_layer_any(ctx, layer, hidden, n_tokens, out, nullptr, static_cast<cudaStream_t>(cuda_stream));
}

int wisp_stack_forward(wisp_ctx* ctx, const void* hidden, int32_t n_tokens, void* hidden_out, void* cuda_stream) {
  int rc = check_forward_args(ctx, 0, ctx ? ctx->cfg.n_layers : 0, hidden, n_tokens, hidden_out);
  if (rc) return rc;
  if (n_tokens == 0) return WISP_OK;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int L = ctx->cfg.n_layers;
  if ((rc = check_dev_err(ctx))) return rc;
  if (ctx->use_fused(n_tokens)) return launch_fused_any(ctx, 0, L, hidden, n_tokens, hidden_out, true, st);
  if (ctx->is_static()) {
    // layer l+1 streams while layer l computes: its copy is queued before layer l's kernels
    const size_t xb = (size_t)n_tokens * ctx->cfg.d_model * ctx->elem;
    CK(cudaMemcpyAsync(ctx->xbuf[0], hidden, xb, cudaMemcpyDeviceToDevice, st));
    int next_streamed = ctx->static_pinned;                          // first layer that needs a copy
    if (next_streamed < L) { rc = static_issue_copy(ctx, next_streamed); if (rc) return rc; }
    for (int l = 0; l < L; ++l) {
      if (l >= ctx->static_pinned && l + 1 < L) { rc = static_issue_copy(ctx, l + 1); if (rc) return rc; }
      rc = forward_layer_static(ctx, l, ctx->xbuf[l & 1], n_tokens, ctx->ybuf, ctx->xbuf[(l + 1) & 1], st, true);
      if (rc) return rc;
    }
    CK(cudaMemcpyAsync(hidden_out, ctx->xbuf[L & 1], xb, cudaMemcpyDeviceToDevice, st));
    return WISP_OK;
  }
  const size_t bytes = (size_t)n_tokens * ctx->cfg.d_model * ctx->elem;
  CK(cudaMemcpyAsync(ctx->xbuf[0], hidden, bytes, cudaMemcpyDeviceToDevice, st));
  auto chain = [&](cudaStream_t s) -> int {
    for (int l = 0; l < L; ++l) {
      int r = forward_layer_any(ctx, l, ctx->xbuf[l & 1], n_tokens, ctx->ybuf, ctx->xbuf[(l + 1) & 1], s);
      if (r) return r;
    }
    return WISP_OK;
  };
  if (ctx->cfg.fetch != WISP_FETCH_MEMCPY && ctx->timing_level == 0 && st != nullptr && n_tokens <= kDecodeMaxTokens && ctx->pf_n == 0) {
    auto it = ctx->graphs.find(n_tokens);
    if (it == ctx->graphs.end()) {
      cudaGraph_t g = nullptr;
      const u64 l0 = ctx->launches;
      CK(cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
      rc = chain(st);
      ctx->graph_nodes[n_tokens] = ctx->launches - l0;
      ctx->launches = l0;
      cudaError_t e = cudaStreamEndCapture(st, &g);
      if (rc) { if (g) cudaGraphDestroy(g); return rc; }
      if (e != cudaSuccess) return fail(ctx, WISP_ECUDA, std::string("graph capture: ") + cudaGetErrorString(e));
      cudaGraphExec_t ge = nullptr;
      e = cudaGraphInstantiate(&ge, g, 0);
      cudaGraphDestroy(g);
      if (e != cudaSuccess) return fail(ctx, WISP_ECUDA, std::string("graph instantiate: ") + cudaGetErrorString(e));
      it = ctx->graphs.emplace(n_tokens, ge).first;
    }
    CK(cudaGraphLaunch(it->second, st));
    ctx->launches += ctx->graph_nodes[n_tokens];
    for (int l = 0; l < L; ++l) ctx->last_T[l] = n_tokens;
    ctx->last_layer = L - 1;
  } else {
    rc = chain(st);
    if (rc) return rc;
  }
  CK(cudaMemcpyAsync(hidden_out, ctx->xbuf[L & 1], bytes, cudaMemcpyDeviceToDevice, st));
  return WISP_OK;
}

int wisp_residual_add(wisp_ctx* ctx, const void* x, const void* y, void* out, int64_t n_elems, void* cuda_stream) {
  if (!ctx || !x || !y || !out || n_elems < 0) return fail(ctx, WISP_EINVAL, "bad argument");
  if (n_elems == 0) return WISP_OK;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const unsigned g = (unsigned)((n_elems + 255) / 256);
  Span sp(ctx, WISP_K_OTHER, st);
  if (ctx->cfg.dtype == WISP_F32)
    residual_add_kernel<float><<<g, 256, 0, st>>>((const float*)x, (const float*)y, (float*)out, (size_t)n_elems);
  else
    residual_add_kernel<__nv_bfloat16><<<g, 256, 0, st>>>((const __nv_bfloat16*)x, (const __nv_bfloat16*)y,
                                                          (__nv_bfloat16*)out, (size_t)n_elems);
  CK(cudaGetLastError());
  return WISP_OK;
}

int wisp_set_split(wisp_ctx* ctx, uint64_t expert_bytes, uint64_t kv_bytes) {
  if (!ctx) return WISP_EINVAL;
  if (ctx->is_static()) return fail(ctx, WISP_ESTATE, "static layer-offload arm: no expert/KV split to move");
  const u64 b = ctx->cfg.kv_block_bytes;
  const u64 Cn64 = std::min<u64>(ctx->cfg.n_experts, expert_bytes / ctx->a_bytes);
  const u64 kap = b ? kv_bytes / b : 0;
  const bool over = expert_bytes > ctx->budget || kv_bytes > ctx->budget - expert_bytes;
  if (over || Cn64 < 1 || kap < ctx->cfg.kv_floor_blocks || kap < ctx->kv_reserved ||
      Cn64 * ctx->a_bytes + kap * b > ctx->budget) {
    ++ctx->failed_resize;   // "If a resize fails, the engine keeps the previous valid split."
    return fail(ctx, WISP_EBUDGET, "split refused: over budget, below the KV floor/reservations, or C < 1");
  }
  const int Cn = (int)Cn64;
  CK(cudaDeviceSynchronize());   // drained barrier
  const bool changed = Cn != ctx->C || kap != ctx->kappa;
  if (Cn != ctx->C) {
    // Free-before-grow: the arena is fixed, so "freeing" the shrinking side is the validation
    // above (the two regions never overlap); a shrink compacts survivors before C changes.
    for (int l = 0; l < ctx->cfg.n_layers; ++l) {
      ResizeArgs a;
      a.E = ctx->cfg.n_experts; a.C_old = ctx->C; a.C_new = Cn; a.policy = ctx->cfg.policy; a.layer = l;
      a.st = layer_state(ctx, l);
      a.moves = ctx->moves; a.n_moves = ctx->moves + 2 * ctx->cfg.n_experts;
      a.trace = ctx->trace; a.trace_ctr = ctx->trace_ctr; a.trace_cap = ctx->trace_cap; a.trace_on = ctx->trace_on;
      residency_resize_kernel<<<1, kPlanThreads>>>(a);
      if (Cn < ctx->C) {
        dim3 g(64, Cn);   // at most Cn moves
        move_slots_kernel<<<g, 256>>>(ctx->moves, a.n_moves, reinterpret_cast<uint4*>(ctx->arena), ctx->Me / 16,
                                      ctx->cfg.n_layers, l);
      }
    }
    CK(cudaGetLastError());
    CK(cudaDeviceSynchronize());
    ctx->C = Cn;
    drop_graphs(ctx);
  }
  ctx->kappa = kap;
  if (changed) ++ctx->resize_count;
  return WISP_OK;
}

int wisp_layer_stats_read(wisp_ctx* ctx, int32_t layer, wisp_layer_stats* out) {
  if (!ctx || !out || layer < 0 || layer >= ctx->cfg.n_layers) return fail(ctx, WISP_EINVAL, "bad argument");
  u64 s[8];
  CK(cudaDeviceSynchronize());
  CK(cudaMemcpy(s, ctx->scal + (size_t)layer * 8, sizeof(s), cudaMemcpyDeviceToHost));
  out->steps = s[1]; out->hits = s[2]; out->misses = s[3]; out->evictions = s[4]; out->references = s[5];
  out->bytes_fetched = s[3] * ctx->Me;
  return WISP_OK;
}

int wisp_stats(wisp_ctx* ctx, wisp_stats_t* out) {
  if (!ctx || !out) return fail(ctx, WISP_EINVAL, "bad argument");
  std::memset(out, 0, sizeof(*out));
  const int L = ctx->cfg.n_layers;
  std::vector<u64> s((size_t)L * 8);
  CK(cudaDeviceSynchronize());
  {
    const int rc = check_dev_err(ctx);
    if (rc) return rc;
  }
  CK(cudaMemcpy(s.data(), ctx->scal, s.size() * sizeof(u64), cudaMemcpyDeviceToHost));
  for (int l = 0; l < L; ++l) {
    out->total.steps += s[l * 8 + 1]; out->total.hits += s[l * 8 + 2]; out->total.misses += s[l * 8 + 3];
    out->total.evictions += s[l * 8 + 4]; out->total.references += s[l * 8 + 5];
  }
  out->total.bytes_fetched = ctx->is_static() ? ctx->static_streamed : out->total.misses * ctx->Me;
  u64 tc[2];
  CK(cudaMemcpy(tc, ctx->trace_ctr, sizeof(tc), cudaMemcpyDeviceToHost));
  harvest_timing(ctx, true);
  out->n_layers = L;
  out->slots_per_layer = ctx->C;
  out->budget_bytes = ctx->budget;
  out->expert_bytes = (u64)ctx->C * ctx->a_bytes;
  out->kv_bytes = ctx->kappa * ctx->cfg.kv_block_bytes;
  out->kv_blocks = ctx->kappa;
  out->kv_blocks_reserved = ctx->kv_reserved;
  out->kv_blocks_peak = ctx->kv_peak;
  out->resize_count = ctx->resize_count;
  out->failed_resize_count = ctx->failed_resize;
  out->trace_dropped = tc[1];
  out->fetch_ns = (u64)(ctx->class_ms[WISP_K_FETCH] * 1e6);
  out->kernel_launches = ctx->launches;
  for (int l = 0; l < L; ++l) out->prefetches += s[l * 8 + 7];
  out->prefetch_bytes = out->prefetches * ctx->Me;
  ctx->kv_peak = ctx->kv_reserved;
  return WISP_OK;
}

int wisp_trace_enable(wisp_ctx* ctx, int32_t on) {
  if (!ctx) return WISP_EINVAL;
  CK(cudaDeviceSynchronize());
  ctx->trace_on = on ? 1 : 0;
  drop_graphs(ctx);   // the flag is a kernel argument baked into captured graphs
  return WISP_OK;
}

int wisp_set_wave_order(wisp_ctx* ctx, int32_t order) {
  if (!ctx) return WISP_EINVAL;
  if (order != WISP_WAVES_ASCENDING && order != WISP_WAVES_HITS_FIRST)
    return fail(ctx, WISP_EINVAL, "wisp_set_wave_order: order must be WISP_WAVES_ASCENDING or WISP_WAVES_HITS_FIRST");
  CK(cudaDeviceSynchronize());
  ctx->wave_order = order;
  drop_graphs(ctx);   // kernel argument baked into captured graphs
  return WISP_OK;
}

int wisp_set_policy(wisp_ctx* ctx, int32_t policy) {
  if (!ctx) return WISP_EINVAL;
  if (policy != WISP_LRU && policy != WISP_LFU) return fail(ctx, WISP_EINVAL, "wisp_set_policy: policy must be WISP_LRU or WISP_LFU");
  CK(cudaDeviceSynchronize());
  ctx->cfg.policy = policy;
  drop_graphs(ctx);   // kernel argument baked into captured graphs
  return WISP_OK;
}

int wisp_set_prefetch(wisp_ctx* ctx, int32_t n_per_layer, double gamma, int32_t window) {
  if (!ctx) return WISP_EINVAL;
  if (ctx->cfg.fetch != WISP_FETCH_ZEROCOPY || n_per_layer < 0 || n_per_layer > kMaxPrefetch || window < 1 || window > kMaxWindow ||
      !(gamma > 0.0 && gamma <= 1.0))
    return fail(ctx, WISP_EINVAL, "wisp_set_prefetch: needs WISP_FETCH_ZEROCOPY, 0 <= n <= 32, 1 <= window <= 4, 0 < gamma <= 1");
  CK(cudaDeviceSynchronize());
  const size_t L = ctx->cfg.n_layers, E = ctx->cfg.n_experts;
  for (void* p : {(void*)ctx->pf_A, (void*)ctx->pf_row, (void*)ctx->pf_rlist, (void*)ctx->pf_rcount, (void*)ctx->pf_copy})
    if (p) cudaFree(p);
  ctx->pf_A = ctx->pf_row = nullptr; ctx->pf_rlist = ctx->pf_rcount = ctx->pf_copy = nullptr;
  ctx->pf_n = 0;
  drop_graphs(ctx);
  if (n_per_layer == 0) return WISP_OK;
  CK(cudaMalloc(&ctx->pf_A, L * window * E * E * sizeof(unsigned)));
  CK(cudaMalloc(&ctx->pf_row, L * window * E * sizeof(unsigned)));
  CK(cudaMalloc(&ctx->pf_rlist, L * E * sizeof(int)));
  CK(cudaMalloc(&ctx->pf_rcount, L * sizeof(int)));
  CK(cudaMalloc(&ctx->pf_copy, L * (1 + 2 * kMaxPrefetch) * sizeof(int)));
  CK(cudaMemset(ctx->pf_A, 0, L * window * E * E * sizeof(unsigned)));
  CK(cudaMemset(ctx->pf_row, 0, L * window * E * sizeof(unsigned)));
  CK(cudaMemset(ctx->pf_rcount, 0, L * sizeof(int)));
  CK(cudaMemset(ctx->pf_copy, 0, L * (1 + 2 * kMaxPrefetch) * sizeof(int)));
  if (!ctx->pf_stream) CK(cudaStreamCreateWithFlags(&ctx->pf_stream, cudaStreamNonBlocking));
  while (ctx->ev_pred.size() < L) {
    cudaEvent_t a, b;
    CK(cudaEventCreateWithFlags(&a, cudaEventDisableTiming));
    CK(cudaEventCreateWithFlags(&b, cudaEventDisableTiming));
    ctx->ev_pred.push_back(a); ctx->ev_copied.push_back(b);
  }
  ctx->pf_pending.assign(L, 0);
  ctx->pf_gpow[0] = 1.0;
  for (int i = 1; i <= kMaxWindow; ++i) ctx->pf_gpow[i] = ctx->pf_gpow[i - 1] * gamma;   // running product, as in oracle/predictor.py
  ctx->pf_window = window;
  ctx->pf_n = n_per_layer;
  return WISP_OK;
}

int wisp_trace_read(wisp_ctx* ctx, wisp_trace_event* buf, uint64_t cap, uint64_t* n_out) {
  if (!ctx || !n_out || (cap && !buf)) return fail(ctx, WISP_EINVAL, "bad argument");
  CK(cudaDeviceSynchronize());
  { const int rc_ = check_dev_err(ctx); if (rc_) return rc_; }
  u64 tc[2];
  CK(cudaMemcpy(tc, ctx->trace_ctr, sizeof(tc), cudaMemcpyDeviceToHost));
  const u64 n = std::min<u64>(cap, tc[0]);
  if (n) CK(cudaMemcpy(buf, ctx->trace, n * sizeof(wisp_trace_event), cudaMemcpyDeviceToHost));
  const u64 rest = tc[0] - n;
  if (rest) {   // keep the undrained tail at the front
    std::vector<wisp_trace_event> tmp(rest);
    CK(cudaMemcpy(tmp.data(), ctx->trace + n, rest * sizeof(wisp_trace_event), cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(ctx->trace, tmp.data(), rest * sizeof(wisp_trace_event), cudaMemcpyHostToDevice));
  }
  tc[0] = rest;
  CK(cudaMemcpy(ctx->trace_ctr, tc, sizeof(u64), cudaMemcpyHostToDevice));
  *n_out = n;
  return WISP_OK;
}

int wisp_last_topk(wisp_ctx* ctx, int32_t layer, int32_t* ids, float* w, int32_t* n_tokens_out) {
  if (!ctx || layer < 0 || layer >= ctx->cfg.n_layers) return fail(ctx, WISP_EINVAL, "bad argument");
  CK(cudaDeviceSynchronize());
  { const int rc_ = check_dev_err(ctx); if (rc_) return rc_; }
  const int T_ = ctx->last_T[layer];
  const size_t off = (size_t)layer * ctx->cfg.max_tokens * ctx->cfg.top_k, n = (size_t)T_ * ctx->cfg.top_k;
  if (ids && n) CK(cudaMemcpy(ids, ctx->ids + off, n * sizeof(int), cudaMemcpyDeviceToHost));
  if (w && n) CK(cudaMemcpy(w, ctx->topw + off, n * sizeof(float), cudaMemcpyDeviceToHost));
  if (n_tokens_out) *n_tokens_out = T_;
  return WISP_OK;
}

int wisp_last_logits(wisp_ctx* ctx, float* z, int32_t n_tokens) {
  if (!ctx || !z || n_tokens < 0 || n_tokens > ctx->cfg.max_tokens) return fail(ctx, WISP_EINVAL, "bad argument");
  CK(cudaDeviceSynchronize());
  { const int rc_ = check_dev_err(ctx); if (rc_) return rc_; }
  if (n_tokens) CK(cudaMemcpy(z, ctx->logits, (size_t)n_tokens * ctx->cfg.n_experts * sizeof(float), cudaMemcpyDeviceToHost));
  return WISP_OK;
}

int wisp_debug_step_routing(wisp_ctx* ctx, int32_t layer, const int32_t* ids, int32_t n_ids) {
  if (!ctx || layer < 0 || layer >= ctx->cfg.n_layers || n_ids < 0 || (n_ids && !ids)) return fail(ctx, WISP_EINVAL, "bad argument");
  if (!ctx->registered[layer]) return fail(ctx, WISP_ESTATE, "layer not registered");
  if (ctx->is_static()) return fail(ctx, WISP_ESTATE, "static layer-offload arm: no pager to drive");
  if (n_ids == 0) return WISP_OK;
  for (int i = 0; i < n_ids; ++i)
    if (ids[i] < 0 || ids[i] >= ctx->cfg.n_experts) return fail(ctx, WISP_EINVAL, "expert id out of range");
  if ((size_t)n_ids > ctx->dbg_ids_cap) {
    if (ctx->dbg_ids) cudaFree(ctx->dbg_ids);
    ctx->dbg_ids = nullptr;
    ctx->dbg_ids_cap = 0;
    CK(cudaMalloc(&ctx->dbg_ids, (size_t)n_ids * sizeof(int)));
    ctx->dbg_ids_cap = n_ids;
  }
  CK(cudaMemcpy(ctx->dbg_ids, ids, (size_t)n_ids * sizeof(int), cudaMemcpyHostToDevice));
  // pair lists are not needed (no FFN): run the plan with build_pairs off by passing the ids directly
  PlanArgs a;
  a.ids = ctx->dbg_ids; a.n_pairs = n_ids; a.E = ctx->cfg.n_experts; a.C = ctx->C; a.policy = ctx->cfg.policy; a.layer = layer;
  a.st = layer_state(ctx, layer); a.plan = ctx->plan; a.host_plan = ctx->host_plan;
  a.trace = ctx->trace; a.trace_ctr = ctx->trace_ctr; a.trace_cap = ctx->trace_cap; a.trace_on = ctx->trace_on;
  a.track = ctx->track; a.build_pairs = n_ids <= std::min<int>(kDecodeMaxTokens, ctx->cfg.max_tokens) * ctx->cfg.top_k ? 1 : 0; a.wave_order = ctx->wave_order;
  residency_plan_kernel<<<1, kPlanThreads>>>(a);
  CK(cudaGetLastError());
  CK(cudaDeviceSynchronize());
  const bool memcpy_path = ctx->cfg.fetch == WISP_FETCH_MEMCPY;
  for (int w = 0; w < ctx->host_plan->n_waves; ++w) {
    int rc = fetch_wave(ctx, layer, w, memcpy_path, nullptr);
    if (rc) return rc;
    CK(cudaDeviceSynchronize());   // wave w+1 may overwrite slots of wave w: keep them serial
  }
  return WISP_OK;
}

int wisp_debug_reset_pool(wisp_ctx* ctx) {
  if (!ctx) return WISP_EINVAL;
  CK(cudaDeviceSynchronize());
  const size_t L = ctx->cfg.n_layers, E = ctx->cfg.n_experts;
  if (!ctx->is_static()) {                                  // (the static arm's maps are the identity and stay)
    CK(cudaMemset(ctx->pi, 0xff, L * E * sizeof(int)));
    CK(cudaMemset(ctx->pi_inv, 0xff, L * E * sizeof(int)));
  }
  ctx->static_streamed = 0;
  if (ctx->pf_n > 0) {                                      // the predictor forgets too: every arm learns from an empty table
    const size_t W = ctx->pf_window;
    CK(cudaMemset(ctx->pf_A, 0, L * W * E * E * sizeof(unsigned)));
    CK(cudaMemset(ctx->pf_row, 0, L * W * E * sizeof(unsigned)));
    CK(cudaMemset(ctx->pf_rcount, 0, L * sizeof(int)));
    ctx->pf_pending.assign(L, 0);
  }
  CK(cudaMemset(ctx->tau, 0, L * E * sizeof(u64)));
  CK(cudaMemset(ctx->freq, 0, L * E * sizeof(u64)));
  CK(cudaMemset(ctx->scal, 0, L * 8 * sizeof(u64)));
  CK(cudaMemset(ctx->last_pos, 0, L * E * sizeof(u64)));
  CK(cudaMemset(ctx->hist, 0, L * (E + 2) * sizeof(u64)));
  std::fill(ctx->host_hist.begin(), ctx->host_hist.end(), 0.0);
  CK(cudaDeviceSynchronize());
  return WISP_OK;
}

int wisp_debug_ffn_launch(wisp_ctx* ctx, int32_t layer, const void* hidden, int32_t n_tokens, void* cuda_stream) {
  if (!ctx || !hidden || layer < 0 || layer >= ctx->cfg.n_layers || n_tokens < 1 || n_tokens > kDecodeMaxTokens ||
      n_tokens > ctx->cfg.max_tokens)
    return fail(ctx, WISP_EINVAL, "bad argument");
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const DecodeGeom g = ctx->dgeom[n_tokens <= 2 ? 0 : 1];
  DecodeSmem sm;
  int rc = decode_smem(ctx, g, n_tokens, ctx->ffn_smem, false, &sm);
  if (rc) return rc;
  DecodeFfnArgs fa{};
  fa.layer_base = ctx->arena + (size_t)layer * ctx->Me; fa.slot_stride = (u64)ctx->cfg.n_layers * ctx->Me;
  fa.blob_bytes = ctx->Me; fa.k = ctx->cfg.top_k;
  fa.partial = ctx->partial; fa.master = nullptr; fa.ticket = ctx->dsync + 1;
  CK(cudaMemsetAsync(ctx->dsync + 1, 0, sizeof(unsigned), st));
  ++ctx->launches;
  if (ctx->f8)
    decode_ffn_kernel<__nv_bfloat16, true><<<ctx->num_sms, kDecThreads, sm.bytes, st>>>(fa, g, ctx->plan, 0, ctx->C, ctx->cfg.n_experts, n_tokens,
                                                                                       static_cast<const __nv_bfloat16*>(hidden), sm.n_slots,
                                                                                       sm.xs_pitch, sm.ring_off);
  else if (ctx->cfg.dtype == WISP_F32)
    decode_ffn_kernel<float, false><<<ctx->num_sms, kDecThreads, sm.bytes, st>>>(fa, g, ctx->plan, 0, ctx->C, ctx->cfg.n_experts, n_tokens,
                                                                                static_cast<const float*>(hidden), sm.n_slots, sm.xs_pitch, sm.ring_off);
  else
    decode_ffn_kernel<__nv_bfloat16, false><<<ctx->num_sms, kDecThreads, sm.bytes, st>>>(fa, g, ctx->plan, 0, ctx->C, ctx->cfg.n_experts, n_tokens,
                                                                                 static_cast<const __nv_bfloat16*>(hidden), sm.n_slots,
                                                                                 sm.xs_pitch, sm.ring_off);
  CK(cudaGetLastError());
  return WISP_OK;
}

int wisp_debug_residency(wisp_ctx* ctx, int32_t layer, int32_t* pi_inv, uint64_t* tau, uint64_t* freq, uint64_t* clock) {
  if (!ctx || layer < 0 || layer >= ctx->cfg.n_layers) return fail(ctx, WISP_EINVAL, "bad argument");
  CK(cudaDeviceSynchronize());
  LayerState s = layer_state(ctx, layer);
  if (pi_inv) CK(cudaMemcpy(pi_inv, s.pi_inv, (size_t)ctx->C * sizeof(int), cudaMemcpyDeviceToHost));
  if (tau) CK(cudaMemcpy(tau, s.tau, (size_t)ctx->C * sizeof(u64), cudaMemcpyDeviceToHost));
  if (freq) CK(cudaMemcpy(freq, s.freq, (size_t)ctx->cfg.n_experts * sizeof(u64), cudaMemcpyDeviceToHost));
  if (clock) CK(cudaMemcpy(clock, s.scal, sizeof(u64), cudaMemcpyDeviceToHost));
  return WISP_OK;
}

int wisp_debug_verify_pool(wisp_ctx* ctx, int32_t layer, int32_t* mismatched_slots) {
  if (!ctx || !mismatched_slots || layer < 0 || layer >= ctx->cfg.n_layers) return fail(ctx, WISP_EINVAL, "bad argument");
  if (!ctx->registered[layer]) return fail(ctx, WISP_ESTATE, "layer not registered");
  if (ctx->is_static()) return fail(ctx, WISP_ESTATE, "static layer-offload arm: no slot pool to verify");
  CK(cudaDeviceSynchronize());
  CK(cudaMemset(ctx->bad_slots, 0, (size_t)ctx->cfg.n_experts * sizeof(int)));
  dim3 g(32, ctx->C);
  verify_pool_kernel<<<g, 256>>>(layer_state(ctx, layer).pi_inv, reinterpret_cast<const uint4*>(ctx->master[layer]),
                                 reinterpret_cast<const uint4*>(ctx->arena), ctx->Me / 16, ctx->cfg.n_layers, layer,
                                 ctx->bad_slots);
  CK(cudaGetLastError());
  std::vector<int> bad(ctx->C);
  CK(cudaMemcpy(bad.data(), ctx->bad_slots, (size_t)ctx->C * sizeof(int), cudaMemcpyDeviceToHost));
  int n = 0;
  for (int v : bad) n += v != 0;
  *mismatched_slots = n;
  return WISP_OK;
}

int wisp_timing_enable(wisp_ctx* ctx, int32_t level) {
  if (!ctx || level < 0 || level > 2) return fail(ctx, WISP_EINVAL, "bad argument");
  ctx->timing_level = level;
  return WISP_OK;
}

int wisp_timing_read(wisp_ctx* ctx, double* ms, uint64_t* launches, int32_t reset) {
  if (!ctx || !ms || !launches) return fail(ctx, WISP_EINVAL, "bad argument");
  CK(cudaDeviceSynchronize());
  harvest_timing(ctx, true);
  if (ctx->fused_layers_timed) {   // phases of the fused decode kernel, stamped with %globaltimer by CTA 0
    u64 ns[kDecPhases + 2];         // + layer calls without a miss, with a miss
    CK(cudaMemcpy(ns, ctx->phase_ns, sizeof(ns), cudaMemcpyDeviceToHost));
    CK(cudaMemset(ctx->phase_ns, 0, sizeof(ns)));
    const int cls[kDecPhases] = {WISP_K_ROUTER, WISP_K_RESIDENCY, WISP_K_OTHER, WISP_K_FFN, WISP_K_FFN_MISS, WISP_K_COMBINE};
    const u64 n_hit = ns[kDecPhases], n_miss = ns[kDecPhases + 1];
    for (int i = 0; i < kDecPhases; ++i) {
      ctx->class_ms[cls[i]] += (double)ns[i] * 1e-6;
      ctx->class_n[cls[i]] += cls[i] == WISP_K_FFN ? n_hit : cls[i] == WISP_K_FFN_MISS ? n_miss : n_hit + n_miss;
    }
    ctx->fused_layers_timed = 0;
  }
  for (int i = 0; i < WISP_N_KERNEL_CLASSES; ++i) { ms[i] = ctx->class_ms[i]; launches[i] = ctx->class_n[i]; }
  if (reset)
    for (int i = 0; i < WISP_N_KERNEL_CLASSES; ++i) { ctx->class_ms[i] = 0.0; ctx->class_n[i] = 0; }
  return WISP_OK;
}

int wisp_kv_reserve(wisp_ctx* ctx, int64_t delta_blocks) {
  if (!ctx) return WISP_EINVAL;
  if (delta_blocks >= 0) {
    if (ctx->kv_reserved + (u64)delta_blocks > ctx->kappa) return fail(ctx, WISP_EBUDGET, "KV pool exhausted");
    ctx->kv_reserved += (u64)delta_blocks;
  } else {
    if ((u64)(-delta_blocks) > ctx->kv_reserved) return fail(ctx, WISP_EBUDGET, "releasing more KV blocks than reserved");
    ctx->kv_reserved -= (u64)(-delta_blocks);
  }
  ctx->kv_peak = std::max(ctx->kv_peak, ctx->kv_reserved);
  return WISP_OK;
}

int wisp_mvwsa_track(wisp_ctx* ctx, int32_t on) {
  if (!ctx) return WISP_EINVAL;
  CK(cudaDeviceSynchronize());
  ctx->track = on ? 1 : 0;
  drop_graphs(ctx);
  return WISP_OK;
}

static int pull_hist(wisp_ctx* ctx) {
  const int L = ctx->cfg.n_layers, E = ctx->cfg.n_experts;
  std::vector<u64> h((size_t)L * (E + 2));
  CK(cudaDeviceSynchronize());
  CK(cudaMemcpy(h.data(), ctx->hist, h.size() * sizeof(u64), cudaMemcpyDeviceToHost));
  CK(cudaMemset(ctx->hist, 0, h.size() * sizeof(u64)));
  for (int l = 0; l < L; ++l)
    for (int i = 0; i < E + 2; ++i) ctx->host_hist[i] += (double)h[(size_t)l * (E + 2) + i];
  return WISP_OK;
}

int wisp_mvwsa_miss_curve(wisp_ctx* ctx, double* m_exp, int32_t n, double decay) {
  if (!ctx || !m_exp || n < 1 || !(decay > 0.0 && decay <= 1.0)) return fail(ctx, WISP_EINVAL, "bad argument");
  int rc = pull_hist(ctx);
  if (rc) return rc;
  const int E = ctx->cfg.n_experts;
  std::vector<double> m = mvwsa::miss_curve(ctx->host_hist, E);
  for (int i = 0; i < n; ++i) m_exp[i] = m[std::min(i, E)];
  if (decay != 1.0)
    for (double& v : ctx->host_hist) v *= decay;
  return WISP_OK;
}

int wisp_mvwsa_propose(wisp_ctx* ctx, const wisp_mvwsa_in* in, uint64_t* expert_bytes, uint64_t* kv_bytes, int32_t* moved) {
  if (!ctx || !in || !expert_bytes || !kv_bytes) return fail(ctx, WISP_EINVAL, "bad argument");
  const u64 b = ctx->cfg.kv_block_bytes;
  if (!b) return fail(ctx, WISP_ESTATE, "no KV accounting (kv_block_bytes == 0)");
  const int E = ctx->cfg.n_experts;
  int64_t c_min = std::max(1, in->c_min), c_max = in->c_max;
  std::vector<double> m;
  if (c_max <= 0 || in->mode == 1) {
    int rc = pull_hist(ctx);
    if (rc) return rc;
    m = mvwsa::miss_curve(ctx->host_hist, E);
  }
  if (c_max <= 0) c_max = std::max<int64_t>(c_min, mvwsa::knee(m, E));
  c_max = std::min<int64_t>(c_max, E);
  int64_t Cn, kap;
  bool mv;
  if (in->mode == 0) {
    const double p = in->kv_peak_blocks == UINT64_MAX ? (double)ctx->kv_peak : (double)in->kv_peak_blocks;
    mvwsa::Split s = mvwsa::live_law(ctx->budget, ctx->a_bytes, b, ctx->cfg.kv_floor_blocks, p, in->headroom, c_min,
                                     c_max, ctx->C, std::max(1, in->dead_zone));
    Cn = s.C; kap = s.kappa; mv = s.moved;
  } else if (in->mode == 1) {
    Cn = mvwsa::configurator(ctx->budget, ctx->a_bytes, b, ctx->cfg.kv_floor_blocks, in->c_exp, in->c_kv, m, in->m_kv,
                             in->m_kv_len, c_min, c_max);
    if (Cn < 0) return fail(ctx, WISP_EBUDGET, "no feasible split above the admission floor");
    kap = (int64_t)((ctx->budget - (u64)Cn * ctx->a_bytes) / b);
    mv = Cn != ctx->C;
  } else {
    return fail(ctx, WISP_EINVAL, "unknown mode");
  }
  *expert_bytes = (u64)Cn * ctx->a_bytes;
  *kv_bytes = (u64)kap * b;
  if (moved) *moved = mv ? 1 : 0;
  return WISP_OK;
}

}  // extern "C"

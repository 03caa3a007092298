/* wisp.h -- C ABI of libwisp: the routed-MoE hot path of WiSP ("Working-Set Paging",
 * arxiv/paper_2606_21868) on one B200 (sm_100a).
 *
 * What the library computes (citations are PAPER.md line numbers; readings Gn are listed in DESIGN.md):
 *   A routed MoE layer forward whose expert weights live in a fixed-budget, slot-indexed VRAM expert
 *   pool while the full expert set stays in pinned host memory (Fig. 1).  Per
 *   layer call: (a1) router GEMV + softmax + top-k; (a2) slot-table residency lookup = Algorithm 1
 *   `WISPLAYER.STEP(R)` with LRU (paper) or LFU (G6) eviction, overflow waves when
 *   |R| > C (G5); (a3) demand fetch of every missing expert from the pinned host master
 *   into its victim slot (Alg. 1 line 6); (a4) SwiGLU expert FFN over slot-indirected weights with a
 *   rank-ordered weighted combine.  The residency requirement is PAPER.md:97: "every expert e in R
 *   must be resident when that layer executes".  Routed experts and KV blocks share ONE pageable
 *   budget B = B_exp + B_kv (Eq. 1); wisp_set_split moves the boundary.
 *
 * Conventions
 *   - Every call returns a wisp_status (0 = OK, negative = error); on error the context is unchanged.
 *     One asynchronous failure exists: if a grid-wide barrier of the fused decode kernel times out (a CTA died),
 *     the kernel abandons the forward, and the NEXT call that synchronises or launches on the context
 *     (wisp_moe_forward, wisp_stack_forward, wisp_stats, wisp_trace_read, wisp_last_topk, wisp_last_logits)
 *     returns WISP_ECUDA once, with wisp_last_error naming it; the outputs of the abandoned forward are invalid.
 *     wisp_last_error() gives a human-readable message for the last failing call on that context.
 *   - "host" / "device" on a pointer says where the memory lives.  The library never takes or returns
 *     framework (torch) types.  `cuda_stream` is a cudaStream_t passed as void* (NULL = default stream).
 *   - One context is used from one thread at a time.  No CPU fallback exists: without a CUDA device
 *     wisp_create fails with WISP_ECUDA.
 *   - Canonical expert blob as the CALLER supplies it (one expert, M_e = 3*d_model*d_ff*sizeof(dtype) bytes,
 *     PAPER.md:102), row-major out x in:  [ gate (d_ff x d_model) | up (d_ff x d_model) | down (d_model x d_ff) ].
 *     wisp_register_host_experts re-tiles it once into the library's in-slot layout (8-row x 16-byte core
 *     matrices, csrc/common.cuh) in its own pinned master; slot bytes == master bytes from then on (the
 *     exactness invariant).
 *   - Arena: one device allocation of `budget_bytes`.  Expert slot s of layer l lives at byte offset
 *     (s*L + l)*M_e  (slot-major, so growing C by one appends a = L*M_e bytes); the KV
 *     pool is the top kappa*b bytes and is modelled as block reservations (BASELINE.json config 5).
 */
#ifndef WISP_H_
#define WISP_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct wisp_ctx wisp_ctx; /* opaque; owned by the library */

typedef enum {
  WISP_OK = 0,
  WISP_EINVAL = -1,   /* bad argument */
  WISP_ENOMEM = -2,   /* host or device allocation failed */
  WISP_ECUDA = -3,    /* CUDA runtime error, or no CUDA device */
  WISP_ESTATE = -4,   /* call not legal in this state (e.g. forward before registration) */
  WISP_EBUDGET = -5   /* split does not fit the budget / floor / reservations */
} wisp_status;

/* WISP_FP8_E4M3 ("The FP8 block-quantized path pages four tensors per expert (the weights and
 * their block scales)"): expert weights are OCP e4m3 codes with one fp32 scale per 128 x 128 block, W[r][c] =
 * e4m3(code[r][c]) * S[r/128][c/128]; hidden states, outputs and the router are bf16 (weight-only quantisation, G29).
 * Canonical fp8 blob (bytes), M_e = 3*d*d_ff + 4 * 3*d*d_ff/16384:
 *   [ W13 codes (2 d_ff x d_model; gate rows, then up rows) | W2 codes (d_model x d_ff) |
 *     S13 fp32 (2 d_ff/128 x d_model/128) | S2 fp32 (d_model/128 x d_ff/128) ]
 * Requires d_model a multiple of 1024 and d_ff a multiple of 256.  The products are exact (fp8 x bf16 on the tensor cores after
 * an exact widening to f16 operands), accumulated in fp32 per 128-wide K block and scaled in fp32. */
typedef enum { WISP_F32 = 0, WISP_BF16 = 1, WISP_FP8_E4M3 = 2 } wisp_dtype;
typedef enum { WISP_LRU = 0, WISP_LFU = 1 } wisp_policy;
/* Miss path (a3): MEMCPY = cudaMemcpyAsync per miss on a dedicated copy stream fenced with events (the
 * host reads the miss list: one host sync per layer call); ZEROCOPY = a device-initiated copy kernel that
 * reads the mapped pinned master (no host round trip; the whole call is stream-ordered); FUSED = no separate
 * copy step in decode: the FFN kernels' TMA producer reads a missing expert's tiles straight from the mapped
 * pinned master, computes on them and writes them into the victim slot (same bytes, same summation order as
 * a hit, so outputs stay byte-identical).  Prefill calls (n_tokens > 8) under FUSED use the ZEROCOPY kernel.
 * STATIC is not a miss path of the method but its COMPARISON ARM: static layer-level offload, "which
 * streams the whole expert layer" (Table 2).  No per-expert residency: the budget holds
 * floor(B / (E*M_e)) - 2 whole layers resident plus a two-layer bounce region; every forward copies ALL E experts of every other
 * layer from the pinned master into the bounce region again (cudaMemcpyAsync on the copy stream, the copy of layer l+1
 * overlapping the compute of layer l inside wisp_stack_forward), then runs the same FFN kernels on it.  Decode-sized calls only
 * (n_tokens <= 8); wisp_set_split, the trace and the pool checks do not apply (ESTATE).  wisp_stats reports the streamed bytes
 * in total.bytes_fetched. */
typedef enum { WISP_FETCH_MEMCPY = 0, WISP_FETCH_ZEROCOPY = 1, WISP_FETCH_FUSED = 2, WISP_FETCH_STATIC = 3 } wisp_fetch;
/* Order in which an overflowing step (|R| > C) is cut into waves of at most C experts (PAPER.md:112 leaves overflow
 * handling to the implementation; G5 / G25).  ASCENDING (default) = ascending expert id.  HITS_FIRST = the
 * members of R resident when the step begins (ascending id) come first, then the faults (ascending id): a resident
 * member is never evicted by an earlier wave of its own step, so the step faults exactly |R \ dom(pi)| times.
 * Steps with |R| <= C are identical under both.  Outputs never depend on the order. */
typedef enum { WISP_WAVES_ASCENDING = 0, WISP_WAVES_HITS_FIRST = 1 } wisp_wave_order;

typedef struct {
  int32_t n_layers;   /* L */
  int32_t n_experts;  /* N (E), 1..1024 */
  int32_t top_k;      /* k, 1..min(E,32) */
  int32_t d_model;    /* multiple of 256 */
  int32_t d_ff;       /* multiple of 256 */
  int32_t max_tokens; /* largest n_tokens passed to wisp_moe_forward (sizes staging buffers) */
  int32_t dtype;      /* wisp_dtype: dtype of weights, hidden and out (WISP_FP8_E4M3: fp8 expert weights, bf16 hidden / out / router) */
  int32_t policy;     /* wisp_policy */
  int32_t fetch;      /* wisp_fetch */
  int32_t ring_stages; /* shared-memory ring depth (parts of <= 32 KiB) of the decode FFN kernels, 2..8; 0 = as many as fit */
  int32_t unit_rows;   /* act rows per decode FFN work unit: multiple of 8 dividing d_ff with d_ff/unit_rows a multiple of 8;
                          0 = library default (16 for bf16 / fp8 models, 8 for fp32).  Outputs are byte-identical across
                          budgets, policies and fetch paths for a GIVEN unit size; changing it regroups the fp32 partial sums. */
  int32_t reserved0;   /* must be 0 */
  uint64_t kv_block_bytes;  /* b: bytes per KV block summed over layers; 0 = no KV accounting */
  uint64_t kv_floor_blocks; /* kappa_min of Eq. 4; wisp_set_split refuses to go below it */
  uint64_t trace_capacity;  /* trace ring capacity in events; 0 = library default (1<<20) */
} wisp_config;

typedef struct {
  uint64_t steps;         /* forwards of this layer with n_tokens > 0 */
  uint64_t references;    /* sum over steps of |R| (distinct experts, G20) */
  uint64_t hits, misses;  /* hits + misses == references */
  uint64_t evictions;
  uint64_t bytes_fetched; /* misses * M_e */
} wisp_layer_stats;

typedef struct {
  wisp_layer_stats total;        /* summed over layers */
  int32_t n_layers;
  int32_t slots_per_layer;       /* C */
  uint64_t budget_bytes;         /* B */
  uint64_t expert_bytes;         /* C * a */
  uint64_t kv_bytes;             /* kappa * b */
  uint64_t kv_blocks;            /* kappa */
  uint64_t kv_blocks_reserved;   /* currently reserved */
  uint64_t kv_blocks_peak;       /* peak reserved since the previous wisp_stats call (p of Eq. 6) */
  uint64_t resize_count;         /* successful wisp_set_split calls that changed C or kappa */
  uint64_t failed_resize_count;  /* refused wisp_set_split calls (state kept) */
  uint64_t trace_dropped;        /* events lost because the ring was full */
  uint64_t fetch_ns;             /* event-timed busy time of the miss path (only while wisp_timing_enable >= 1) */
  uint64_t kernel_launches;      /* library kernels launched so far (graph replays count their kernel nodes) */
  uint64_t prefetches;           /* experts brought in speculatively (wisp_set_prefetch); not counted as misses */
  uint64_t prefetch_bytes;       /* prefetches * M_e: host-link bytes spent on speculation */
} wisp_stats_t;

/* Kernel classes of wisp_timing_read.  Decode (n_tokens <= 8): ROUTER = logits + top-k, RESIDENCY = Algorithm 1, FFN = the fused
 * gate/up/SwiGLU/down stream of layer calls without a miss (inside the fused kernel: including the grid barrier that ends it),
 * FFN_MISS = the same for layer calls with >= 1 miss, COMBINE = ordered combine + residual + next layer's partial logits.
 * Prefill: ROUTER, TOPK, RESIDENCY, FETCH, PREFILL_GATE_UP, PREFILL_DOWN, COMBINE, OTHER (gather, work lists). */
enum { WISP_K_ROUTER = 0, WISP_K_TOPK = 1, WISP_K_RESIDENCY = 2, WISP_K_FETCH = 3, WISP_K_FFN = 4, WISP_K_FFN_MISS = 5,
       WISP_K_COMBINE = 6, WISP_K_PREFILL_GATE_UP = 7, WISP_K_PREFILL_DOWN = 8, WISP_K_OTHER = 9,
       WISP_N_KERNEL_CLASSES = 10 };

/* kind: 0 hit, 1 miss, 2 resize-drop, 3 resize-move (for a move `evicted` carries the source slot), 4 speculative prefetch
 * (emitted between the events of layer l and those of layer l+1, best-scoring expert first; `step` = the target layer's next step).
 * Events of one wave are emitted in wave order (ascending expert id; under WISP_WAVES_HITS_FIRST an overflowing step
 * lists residents, then faults, each ascending); waves in order; layers/steps in call order. */
typedef struct {
  uint64_t step;   /* per-layer step counter (0-based) */
  uint32_t layer;
  uint32_t wave;
  int32_t expert;
  int32_t slot;
  int32_t evicted; /* -1 none */
  uint32_t kind;
} wisp_trace_event;

/* Inputs of the MV-WSA proposal (PAPER.md:126-169 and App. B).  mode 0 = live law, Eq. 6-8
 * (PAPER.md:353-363): kappa~ = max(kappa_min, ceil((1+h)p)); C~ = clip(floor((B-kappa~ b)/a), C_min, C_max);
 * kappa~ <- floor((B - C~ a)/b); moves smaller than `dead_zone` experts are suppressed.
 * mode 1 = configurator, Eq. 2-5: argmin over C of c_exp*m_exp(C) + c_kv*m_kv(kappa(C))
 * subject to the admission floor, with m_exp taken from the library's decayed reuse-distance histograms
 * and m_kv given by the caller as a table. */
typedef struct {
  int32_t mode;
  int32_t c_min, c_max;      /* clip range for C; c_max <= 0 means "knee of the measured miss curve" (G11) */
  int32_t dead_zone;         /* Delta, experts */
  double headroom;           /* h */
  uint64_t kv_peak_blocks;   /* p; UINT64_MAX = use the peak recorded by wisp_kv_reserve */
  double c_exp;              /* cost of one expert miss  (M_e * t_byte), seconds */
  double c_kv;               /* cost of one KV miss unit (beta * b_tok), seconds */
  const double* m_kv;        /* host, m_kv[kappa] for kappa = 0..m_kv_len-1 (last value extends); may be NULL */
  uint64_t m_kv_len;
} wisp_mvwsa_in;

/* ---- mandated entry points (BASELINE.json north_star) ------------------------------------------- */

/* Create a context with a pageable budget of `budget_bytes` (B).  Allocates the arena and all
 * per-layer state.  Initial split: kv = kv_floor_blocks*b, experts = the rest (C = min(E, floor(./a))).
 * Errors: EINVAL (shape), EBUDGET (fewer than 1 slot per layer fits), ENOMEM, ECUDA.  *out receives the
 * context; destroy with wisp_destroy. */
int wisp_create(uint64_t budget_bytes, const wisp_config* cfg, wisp_ctx** out);
int wisp_destroy(wisp_ctx* ctx);

/* Register one layer's full expert set: the "CPU master W^cpu" of Algorithm 1.
 *   experts     host, E canonical blobs, E*M_e bytes, in cfg.dtype.
 *   router_w    host, [E, d_model] row-major in cfg.dtype (bf16 for WISP_FP8_E4M3).
 *   router_bias host, [E] fp32, or NULL (zeros).
 * The library COPIES all three (experts into its own pinned, device-mapped host memory; router into
 * device memory, which is a fixed cost outside B); the caller may free its buffers on return.
 * Re-registering a layer is an error (ESTATE).  The pool starts empty (cold). */
int wisp_register_host_experts(wisp_ctx* ctx, int32_t layer, const void* experts, const void* router_w,
                               const float* router_bias);

/* One forward of one MoE layer = one "step" of that layer's clock (Alg. 1).
 *   hidden  device, [n_tokens, d_model] row-major, cfg.dtype, 16-byte aligned.
 *   out     device, [n_tokens, d_model], cfg.dtype; out[t] = sum_i w[t,i] * FFN_{ids[t,i]}(hidden[t]).
 * Work is enqueued on `cuda_stream`; `out` is valid once the caller synchronises that stream.  With
 * WISP_FETCH_MEMCPY the call blocks the host until the layer's routing is known.  n_tokens == 0 is a
 * no-op (no tick).  Errors: EINVAL (layer, n_tokens > max_tokens), ESTATE (layer not registered). */
int wisp_moe_forward(wisp_ctx* ctx, int32_t layer, const void* hidden, int32_t n_tokens, void* out,
                     void* cuda_stream);

/* Move the expert<->KV boundary: C = min(E, floor(expert_bytes / a)),
 * kappa = floor(kv_bytes / b).  Legal only between forwards (the "drained barrier"); synchronises the
 * device.  Shrink keeps the C~ best residents by the policy key and compacts them into slots < C~
 * (device-to-device moves, byte-equal to the paper's re-page); grow adds empty slots.  Transactional:
 * EBUDGET (and failed_resize_count++) when expert_bytes + kv_bytes > B, C~ < 1, kappa~ < kv_floor_blocks
 * or kappa~ < blocks currently reserved; the previous split then stays in force. */
int wisp_set_split(wisp_ctx* ctx, uint64_t expert_bytes, uint64_t kv_bytes);

/* Totals and the current split.  Synchronises the device.  Resets kv_blocks_peak to the current level. */
int wisp_stats(wisp_ctx* ctx, wisp_stats_t* out);

/* ---- whole-token helpers (same kernels; O3 semantics of DESIGN.md) ------------------------------- */

/* x_0 = hidden; for l = 0..L-1: y_l = MoE_l(x_l); x_{l+1} = x_l + y_l (add in fp32 on the model-dtype
 * values, stored in cfg.dtype); hidden_out = x_L.  Each layer ticks once.  With WISP_FETCH_ZEROCOPY the
 * chain is replayed from a CUDA graph cached per n_tokens.  hidden/hidden_out: device [n_tokens, d_model]. */
int wisp_stack_forward(wisp_ctx* ctx, const void* hidden, int32_t n_tokens, void* hidden_out,
                       void* cuda_stream);
/* out = x + y elementwise with the rounding stated above (device pointers, n_elems elements of cfg.dtype). */
int wisp_residual_add(wisp_ctx* ctx, const void* x, const void* y, void* out, int64_t n_elems,
                      void* cuda_stream);

/* ---- parity / test surface ------------------------------------------------------------------------ */

int wisp_layer_stats_read(wisp_ctx* ctx, int32_t layer, wisp_layer_stats* out);
/* Trace ring: when on, every reference / resize action appends one wisp_trace_event. */
int wisp_trace_enable(wisp_ctx* ctx, int32_t on);
/* Select the overflow wave order (wisp_wave_order) for all later forwards.  Synchronises the device; residency state,
 * counters and slot contents are kept.  Errors: EINVAL (NULL ctx or unknown order; state unchanged). */
int wisp_set_wave_order(wisp_ctx* ctx, int32_t order);
/* Select the eviction policy (wisp_policy) for all later forwards; tau and f are kept (both are maintained under either
 * policy), so a switch is usually followed by wisp_debug_reset_pool.  Synchronises.  Errors: EINVAL. */
int wisp_set_policy(wisp_ctx* ctx, int32_t policy);
/* Speculative expert prefetch driven by the online co-activation predictor of the paper's App. E (Section 4,
 * PAPER.md:175-189 reports that it LOWERS single-stream decode throughput: the copies compete with demand traffic for the same
 * link).  After layer l has routed, the n_per_layer best-scoring absent experts of layer l+1 (score s_{l+1}(e') = sum over the
 * `window` previous layers of gamma^dist * sum_{e in R_l} P(e'|e), tables learned online from an empty start) are copied from the
 * pinned master on a side stream into the victim slots of layer l+1 (increasing policy key; G27) while layer l's FFN
 * runs.  Split decode form only: EINVAL unless cfg.fetch == WISP_FETCH_ZEROCOPY, 0 <= n_per_layer <= 32, 1 <= window <= 4,
 * 0 < gamma <= 1.  n_per_layer = 0 switches it off; the tables are cleared on every call.  Outputs never change.  Synchronises. */
int wisp_set_prefetch(wisp_ctx* ctx, int32_t n_per_layer, double gamma, int32_t window);
/* Drain up to `cap` events into host `buf` (oldest first); *n_out = number written.  Synchronises. */
int wisp_trace_read(wisp_ctx* ctx, wisp_trace_event* buf, uint64_t cap, uint64_t* n_out);
/* Routing of the most recent forward of `layer`: host ids [n_tokens, k] (rank order) and w [n_tokens, k].
 * *n_tokens_out (may be NULL) receives that forward's n_tokens.  Either array may be NULL.  Synchronises. */
int wisp_last_topk(wisp_ctx* ctx, int32_t layer, int32_t* ids, float* w, int32_t* n_tokens_out);
/* Router logits of the most recent forward overall: host z [n_tokens, E] fp32.  Synchronises. */
int wisp_last_logits(wisp_ctx* ctx, float* z, int32_t n_tokens);
/* The router step of one layer (a1: logits, top-k ids in (z desc, id asc) order, softmax over the selected k) for a small token
 * batch WITHOUT any allocation -- for callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses
 * that forbid it).  No context: the caller passes every input and output; the only scratch (the 2^-32 fixed-point int64 logit
 * accumulators of the decode path) is a file-scope device array of 8192 words = 64 KiB that every GPU loading the library holds
 * until exit.  Same arithmetic as the context's decode path, so the results equal wisp_last_logits / wisp_last_topk bit for bit.
 *   hidden       device, [n_tokens, d_model] row-major, `dtype` (WISP_F32 or WISP_BF16)
 *   router_w     device, [n_experts, d_model] row-major, `dtype`;  router_bias  device, [n_experts] fp32, or NULL (zeros)
 *   logits       device, [n_tokens, n_experts] fp32 out, or NULL;  ids  device, [n_tokens, top_k] int32 out;  w  device, [n_tokens, top_k] fp32 out
 * Limits: n_tokens * n_experts <= 8192 (else WISP_EINVAL, with the reason on stderr), n_experts <= 1024, top_k <= min(E, 32),
 * d_model a multiple of 16.  Calls no cudaMalloc / cudaFree; work is queued on `cuda_stream` (memset + two kernels), not synchronised.
 * All calls share the scratch array (each clears the words it uses first): calls that overlap on the GPU race -- serialise them. */
int wisp_route_noalloc(const void* hidden, const void* router_w, const float* router_bias, int32_t n_tokens, int32_t n_experts,
                       int32_t d_model, int32_t top_k, int32_t dtype, float* logits, int32_t* ids, float* w, void* cuda_stream);
/* Drive the pager with a given routed-id list (host, n_ids ids, repeats allowed): runs the residency
 * lookup and the demand fetch of one step of `layer`, no router and no FFN.  Synchronises. */
int wisp_debug_step_routing(wisp_ctx* ctx, int32_t layer, const int32_t* ids, int32_t n_ids);
/* Empty the expert pool of every layer and zero the paging state and counters (pi, pi^-1, tau, f, clock, steps, hits, misses,
 * evictions, references; reuse-distance histograms): the context is as cold as after registration.  Slot contents, the split
 * and KV reservations are kept.  Measurement / verification helper: every timed arm starts from this state.  Synchronises. */
int wisp_debug_reset_pool(wisp_ctx* ctx);
/* FFN-only replay (microbenchmark m1): launches the decode FFN kernel for wave 0 of the plan left by the most recent
 * wisp_debug_step_routing(layer, ids) -- ids given in (token, rank) order, n_tokens*top_k of them, every expert resident after
 * that call -- on `hidden` (device, [n_tokens, d_model]); no router, no lookup, no combine.  n_tokens <= 8.  Asynchronous. */
int wisp_debug_ffn_launch(wisp_ctx* ctx, int32_t layer, const void* hidden, int32_t n_tokens, void* cuda_stream);
/* Residency state of `layer`: host pi_inv [C] (expert per slot, -1 empty), tau [C], freq [E], *clock.
 * Any pointer may be NULL.  Synchronises. */
int wisp_debug_residency(wisp_ctx* ctx, int32_t layer, int32_t* pi_inv, uint64_t* tau, uint64_t* freq,
                         uint64_t* clock);
/* Exactness invariant check: compares every occupied slot of `layer` byte for byte with
 * the host master of the expert it claims to hold; *mismatched_slots = number of slots that differ. */
int wisp_debug_verify_pool(wisp_ctx* ctx, int32_t layer, int32_t* mismatched_slots);
/* CUDA-event timing of the library's own launches, on the stream each is launched on.  level 0 = off,
 * 1 = the miss path only (WISP_K_FETCH; also summed into wisp_stats.fetch_ns), 2 = every kernel class.  While
 * level > 0 wisp_stack_forward does not replay CUDA graphs.  wisp_timing_read: host ms[WISP_N_KERNEL_CLASSES]
 * (summed event-to-event milliseconds) and launches[WISP_N_KERNEL_CLASSES] (timed spans); reset != 0 zeroes
 * the totals after the read.  Synchronises. */
int wisp_timing_enable(wisp_ctx* ctx, int32_t level);
int wisp_timing_read(wisp_ctx* ctx, double* ms, uint64_t* launches, int32_t reset);

/* ---- KV reservations and MV-WSA (CPU side) ----------------------------- */

/* Reserve (delta > 0) or release (delta < 0) KV blocks; EBUDGET if it would exceed kappa or go below 0. */
int wisp_kv_reserve(wisp_ctx* ctx, int64_t delta_blocks);
/* Propose a split (does not apply it): see wisp_mvwsa_in.  Outputs are byte counts that wisp_set_split
 * accepts: expert_bytes = C~*a, kv_bytes = kappa~*b.  *moved (may be NULL) = 0 when the dead zone held. */
int wisp_mvwsa_propose(wisp_ctx* ctx, const wisp_mvwsa_in* in, uint64_t* expert_bytes, uint64_t* kv_bytes,
                       int32_t* moved);
/* Expert miss curve from the library's reuse-distance histograms: host m_exp[0..n-1],
 * m_exp[C] = (decayed) number of references with stack distance > C, summed over layers.  `decay` in
 * (0,1] multiplies all bins AFTER the read ("decayed"); 1.0 = leave unchanged.
 * Histograms are fed from the routing of every forward while tracking is on (wisp_mvwsa_track). */
int wisp_mvwsa_miss_curve(wisp_ctx* ctx, double* m_exp, int32_t n, double decay);
int wisp_mvwsa_track(wisp_ctx* ctx, int32_t on);

const char* wisp_last_error(wisp_ctx* ctx);
/* Library build info, e.g. "libwisp sm_100a ..." (static string). */
const char* wisp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* WISP_H_ */

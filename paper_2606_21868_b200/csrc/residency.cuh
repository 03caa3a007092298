// residency.cuh -- (a2) slot-table residency lookup = Algorithm 1 WISPLAYER.STEP(R)
// run ON THE DEVICE (the paper runs it in Python on the host and names that the overhead to remove,
// PAPER.md:444), plus the resize of a7.  Integer work only; one CTA per layer call.
//
// Readings: G1 M = R \ dom(pi); G2 ties -> lower slot; G3 M ascending id <-> U in key order;
// G4 empty slots (tau = 0) first; G5 waves of <= C ascending ids; G6 LFU key (f, tau, slot), empty f = -1;
// G24 one tick per wave; G25 wave order: WISP_WAVES_HITS_FIRST lists R as (residents at step start, ascending id)
// then (faults, ascending id) when |R| > C (overflow handling is an implementation detail).
#pragma once
#include "common.cuh"

namespace wisp {

constexpr int kPlanThreads = 1024;

struct PlanArgs {
  const int* ids;   // [n_pairs] routed expert ids (t*k + rank order)
  int n_pairs;
  int E, C, policy, layer;
  LayerState st;
  PlanPtrs plan;
  HostPlan* host_plan;            // nullable (MEMCPY path)
  wisp_trace_event* trace;        // ring
  u64* trace_ctr;                 // [0] count, [1] dropped
  u64 trace_cap;
  int trace_on;
  int track;                      // MV-WSA reuse-distance tracking
  int build_pairs;                // build pair_list here (small n_pairs) or leave it to group_pairs_kernel
  int wave_order;                 // wisp_wave_order (G25)
};

// ---- Algorithm 1 as a device function, usable by a standalone CTA (NT = 1024 threads) and by every CTA of the
// persistent decode kernel (NT = 256 consumer threads, all CTAs compute the same plan, one of them is the writer).
// NT = participating threads (threadIdx.x < NT) = capacity in experts (E <= NT); `bar` = named barrier id for them.
template <int NT>
struct PlanShared {
  unsigned bitmap[NT / 32];
  int cnt[NT];
  int R[NT];              // sorted distinct routed ids
  int pi[NT];
  int pinv[NT];
  u64 tau[NT];
  u64 freq[NT];
  u64 kf[NT];             // LFU component of the victim key per slot (also scratch of the MV-WSA tracking pass)
  unsigned char inw[NT], elig[NT];
  int victim[NT];
  int ws[NT / 32 + 1];
  u64 scal[8];            // the layer's scalars as loaded (clock, step, hits, misses, evictions, references, position)
  u64 clock;
  int evict;
};

template <int NT>
__device__ __forceinline__ void plan_sync(int bar) { asm volatile("bar.sync %0, %1;" ::"r"(bar), "n"(NT) : "memory"); }

// exclusive scan over the NT participating threads; ws = NT/32 + 1 ints of scratch
template <int NT>
__device__ __forceinline__ int block_excl_scan(int v, int* ws, int& total, int bar) {
  constexpr int NW = NT / 32;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int n = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += n;
  }
  if (lane == 31) ws[wid] = inc;
  plan_sync<NT>(bar);
  if (wid == 0) {
    int s = lane < NW ? ws[lane] : 0, si = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int n = __shfl_up_sync(0xffffffffu, si, o);
      if (lane >= o) si += n;
    }
    if (lane < NW) ws[lane] = si - s;
    if (lane == 31) ws[NW] = si;
  }
  plan_sync<NT>(bar);
  total = ws[NW];
  int r = inc - v + ws[wid];
  plan_sync<NT>(bar);
  return r;
}

// victim order: LRU (tau, slot); LFU (f+1 or 0 for empty, tau, slot)   -- ascending
__device__ __forceinline__ bool key_less(u64 fa, u64 ta, int sa, u64 fb, u64 tb, int sb) {
  if (fa != fb) return fa < fb;
  if (ta != tb) return ta < tb;
  return sa < sb;
}

// pi, pi^-1, tau, f, clock of this layer -> shared memory.  The caller synchronises before plan_compute.
template <int NT>
__device__ __forceinline__ void plan_load(PlanShared<NT>& sh, const LayerState& st, int E, int C) {
  const int tid = threadIdx.x;
  if (tid < E) { sh.pi[tid] = st.pi[tid]; sh.freq[tid] = st.freq[tid]; }
  if (tid < C) { sh.pinv[tid] = st.pi_inv[tid]; sh.tau[tid] = st.tau[tid]; }
  if (tid < 8) sh.scal[tid] = st.scal[tid];
  if (tid == 0) sh.clock = st.scal[0];
}

// One WISPLAYER.STEP(R) (all waves) on the state in `sh`; the plan goes to a.plan (global or shared pointers).
// writer: this CTA also writes the state back, counts, traces and feeds the MV-WSA histograms.
template <int NT>
__device__ __forceinline__ void plan_compute(const PlanArgs& a, PlanShared<NT>& sh, bool writer, int bar) {
  const int tid = threadIdx.x;
  const int E = a.E, C = a.C;
  if (tid < NT / 32) sh.bitmap[tid] = 0u;
  if (tid < E) sh.cnt[tid] = 0;
  if (tid == 0) sh.evict = 0;
  plan_sync<NT>(bar);

  // ---- R = set of routed ids; per-expert pair counts ----
  for (int p = tid; p < a.n_pairs; p += NT) {
    int e = a.ids[p];
    atomicOr(&sh.bitmap[e >> 5], 1u << (e & 31));
    atomicAdd(&sh.cnt[e], 1);
  }
  plan_sync<NT>(bar);
  int total = 0;
  {
    const int present = (tid < E) ? ((sh.bitmap[tid >> 5] >> (tid & 31)) & 1) : 0;
    int pos = block_excl_scan<NT>(present, sh.ws, total, bar);
    if (present) sh.R[pos] = tid;
  }
  const int nR = total;
  {
    int tot2;
    int off = block_excl_scan<NT>(tid < E ? sh.cnt[tid] : 0, sh.ws, tot2, bar);
    if (tid < E) { a.plan.exp_offset[tid] = off; a.plan.exp_count[tid] = sh.cnt[tid]; }
    if (tid == 0) a.plan.exp_offset[E] = tot2;
    if (a.build_pairs && tid < a.n_pairs) {
      // stable grouping for small n_pairs: rank among lower-indexed pairs of the same expert
      const int e = a.ids[tid];
      int r = 0;
      for (int q = 0; q < tid; ++q) r += (a.ids[q] == e);
      sh.victim[tid] = r;   // borrowed as scratch (n_pairs <= NT in this mode)
    }
  }
  plan_sync<NT>(bar);
  if (a.build_pairs && tid < a.n_pairs) {
    const int e = a.ids[tid];
    a.plan.pair_list[a.plan.exp_offset[e] + sh.victim[tid]] = tid;   // exp_offset written by thread e above
  }
  plan_sync<NT>(bar);

  // ---- MV-WSA reuse-distance tracking: stack distance of every reference ----
  if (writer && a.track && nR > 0) {
    u64* s_last = sh.kf;
    if (tid < E) s_last[tid] = a.st.last_pos[tid];
    plan_sync<NT>(bar);
    const u64 base = sh.scal[6];     // linear position counter of this layer
    if (tid < nR) {
      const int e = sh.R[tid];
      const u64 mine = s_last[e];
      int bin;
      if (mine == 0) {
        bin = E + 1;                 // first reference: infinite distance
      } else {
        int dist = 1 + tid;          // e itself + the tid lower ids of this step (referenced just before)
        for (int o = 0; o < E; ++o) {
          if (o == e) continue;
          const bool in_step_before = ((sh.bitmap[o >> 5] >> (o & 31)) & 1) && o < e;
          if (!in_step_before && s_last[o] > mine) ++dist;
        }
        bin = dist > E ? E + 1 : dist;
      }
      atomicAdd(&a.st.hist[bin], 1ull);
    }
    plan_sync<NT>(bar);
    if (tid < nR) a.st.last_pos[sh.R[tid]] = base + 1 + tid;
    if (tid == 0) a.st.scal[6] = base + nR;
    plan_sync<NT>(bar);
  }

  // ---- G25: hits-first listing of R (only when the step overflows; one wave gives the same plan either way) ----
  if (a.wave_order == WISP_WAVES_HITS_FIRST && nR > C) {
    const int e = tid < nR ? sh.R[tid] : -1;
    const int res = (e >= 0 && sh.pi[e] >= 0) ? 1 : 0;
    int n_res;
    const int ri = block_excl_scan<NT>(res, sh.ws, n_res, bar);   // ends with a barrier: every R[tid] has been read
    if (e >= 0) sh.R[res ? ri : n_res + (tid - ri)] = e;
    plan_sync<NT>(bar);
  }

  // ---- Algorithm 1 per wave ----
  const int n_waves = (nR + C - 1) / C;
  const u64 step_no = sh.scal[1];
  bool trace_ok = false;
  u64 trace_base = 0;
  if (writer && a.trace_on) {
    trace_base = a.trace_ctr[0];
    trace_ok = trace_base + (u64)nR <= a.trace_cap;
  }
  int hits_total = 0, miss_total = 0;
  for (int wv = 0; wv < n_waves; ++wv) {
    const int lo = wv * C;
    const int nw = min(C, nR - lo);
    if (tid < E) sh.inw[tid] = 0;
    plan_sync<NT>(bar);
    int e = -1, is_miss = 0;
    if (tid < nw) { e = sh.R[lo + tid]; sh.inw[e] = 1; is_miss = sh.pi[e] < 0; }
    plan_sync<NT>(bar);
    int n_miss;
    const int mi = block_excl_scan<NT>(is_miss, sh.ws, n_miss, bar);       // line 2: M = R \ dom(pi), ascending id
    // line 3: U = {s : pi^-1(s) not in R} in increasing key
    if (tid < C) {
      const int occ = sh.pinv[tid];
      sh.elig[tid] = (occ < 0) || !sh.inw[occ];
      sh.kf[tid] = (a.policy == WISP_LFU) ? (occ < 0 ? 0ull : sh.freq[occ] + 1ull) : 0ull;
    }
    plan_sync<NT>(bar);
    if (tid < C && sh.elig[tid] && n_miss > 0) {
      const u64 kf = sh.kf[tid], kt = sh.tau[tid];
      int rank = 0;
      for (int o = 0; o < C; ++o)
        if (sh.elig[o] && key_less(sh.kf[o], sh.tau[o], o, kf, kt, tid)) ++rank;
      if (rank < n_miss) sh.victim[rank] = tid;
    }
    plan_sync<NT>(bar);
    // lines 4-8: assign, (the copy happens in the fetch step), update the maps
    int slot = -1, old = -1;
    if (tid < nw) {
      if (is_miss) {
        slot = sh.victim[mi];
        old = sh.pinv[slot];
        if (old >= 0) { sh.pi[old] = -1; atomicAdd(&sh.evict, 1); }
        sh.pi[e] = slot;
        sh.pinv[slot] = e;
      } else {
        slot = sh.pi[e];
      }
    }
    if (tid == 0) sh.clock += 1;                                   // line 9: c <- c + 1
    plan_sync<NT>(bar);
    if (tid < nw) {
      sh.tau[slot] = sh.clock;                                     // tau[pi(e)] <- c
      sh.freq[e] += 1ull;
      const int idx = lo + tid;
      a.plan.entry_expert[idx] = e;
      a.plan.entry_slot[idx] = slot;
      a.plan.entry_miss[idx] = is_miss;
      if (writer && a.host_plan) {
        a.host_plan->entry_expert[idx] = e;
        a.host_plan->entry_slot[idx] = slot;
        a.host_plan->entry_miss[idx] = is_miss;
      }
      if (trace_ok) {
        wisp_trace_event ev;
        ev.step = step_no; ev.layer = (uint32_t)a.layer; ev.wave = (uint32_t)wv;
        ev.expert = e; ev.slot = slot; ev.evicted = old; ev.kind = is_miss ? 1u : 0u;
        a.trace[trace_base + idx] = ev;
      }
    }
    hits_total += nw - n_miss;
    miss_total += n_miss;
    plan_sync<NT>(bar);
  }
  if (tid == 0) { a.plan.hdr[0] = n_waves; a.plan.hdr[1] = nR; a.plan.hdr[2] = miss_total; a.plan.hdr[3] = a.n_pairs; }
  // decode path: unit order of every wave (misses first, each group in wave order) and the inverse pair permutation
  if (a.plan.unit_entry != nullptr && tid < nR) {
    const int lo = (tid / C) * C, nw = min(C, nR - lo);
    const int mine = a.plan.entry_miss[tid];
    int miss_before = 0, hit_before = 0, miss_all = 0;
    for (int o = 0; o < nw; ++o) {
      const int m = a.plan.entry_miss[lo + o];
      miss_all += m;
      if (lo + o < tid) { miss_before += m; hit_before += 1 - m; }
    }
    a.plan.unit_entry[lo + (mine ? miss_before : miss_all + hit_before)] = tid;
  }
  if (a.plan.pair_pos != nullptr && a.build_pairs && tid < a.n_pairs) a.plan.pair_pos[a.plan.pair_list[tid]] = tid;

  // ---- write back ----
  if (writer) {
    if (tid < E) { a.st.pi[tid] = sh.pi[tid]; a.st.freq[tid] = sh.freq[tid]; }
    if (tid < C) { a.st.pi_inv[tid] = sh.pinv[tid]; a.st.tau[tid] = sh.tau[tid]; }
    if (tid == 0) {
      if (a.host_plan) {
        a.host_plan->n_ref = nR; a.host_plan->n_miss = miss_total; a.host_plan->n_pairs = a.n_pairs;
        __threadfence_system();
        a.host_plan->n_waves = n_waves;
      }
      a.st.scal[0] = sh.clock;                    // stores only: the old values were loaded by plan_load
      if (nR > 0) a.st.scal[1] = step_no + 1;
      a.st.scal[2] = sh.scal[2] + (u64)hits_total;
      a.st.scal[3] = sh.scal[3] + (u64)miss_total;
      a.st.scal[4] = sh.scal[4] + (u64)sh.evict;
      a.st.scal[5] = sh.scal[5] + (u64)nR;
      if (a.trace_on) {
        if (trace_ok) a.trace_ctr[0] = trace_base + (u64)nR;
        else a.trace_ctr[1] += (u64)nR;
      }
    }
  }
  plan_sync<NT>(bar);
}

// Hit fast path of WISPLAYER.STEP(R) for decode-sized calls, run by ONE warp (lanes of warp 0 of the caller): when every
// member of R is already resident and |R| <= C, Algorithm 1 has no fault to assign (lines 2-8 are empty) and the step is
// just the tick of line 9: c <- c+1, tau[pi(e)] <- c, f[e] += 1 for e in R (G24).  Builds the same plan
// plan_compute would (entries in ascending id, pairs grouped by expert) and returns true; returns false -- touching nothing
// but its scratch -- when the step has a fault, overflows, is being tracked for MV-WSA or has more than 64 pairs, and the
// caller then runs plan_compute.  `sh` holds the layer's state as loaded by plan_load.
template <int NT>
__device__ __forceinline__ bool plan_fast_warp(const PlanArgs& a, PlanShared<NT>& sh, bool writer, int lane) {
  const int E = a.E, n_pairs = a.n_pairs;
  if (a.track || n_pairs > 64 || E > NT) return false;
  // Lane l holds pairs l and l + 32.  One pass of warp shuffles gives every pair its position in the expert-sorted pair
  // order (pairs ordered by (expert id, pair index)), its expert's pair count and whether it is the first pair of its expert.
  const int n_hi = n_pairs > 32 ? n_pairs - 32 : 0;
  int e[2] = {lane < n_pairs ? a.ids[lane] : 0x7fffffff, lane < n_hi ? a.ids[lane + 32] : 0x7fffffff};
  int pos[2] = {0, 0}, cnt[2] = {0, 0};
  bool first[2] = {true, true};
  const int n_lo = min(n_pairs, 32);
  for (int q = 0; q < n_lo; ++q) {
    const int eq = __shfl_sync(0xffffffffu, e[0], q);
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int me = lane + 32 * h;
      pos[h] += (eq < e[h]) || (eq == e[h] && q < me);
      cnt[h] += (eq == e[h]);
      first[h] = first[h] && !(eq == e[h] && q < me);
    }
  }
  for (int q = 0; q < n_hi; ++q) {
    const int eq = __shfl_sync(0xffffffffu, e[1], q);
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int me = lane + 32 * h;
      pos[h] += (eq < e[h]) || (eq == e[h] && q + 32 < me);
      cnt[h] += (eq == e[h]);
      first[h] = first[h] && !(eq == e[h] && q + 32 < me);
    }
  }
  const bool live[2] = {lane < n_pairs, lane < n_hi};
  // entry index of an expert = number of distinct smaller ids = first-pairs that sort before it
  const unsigned lead0 = __ballot_sync(0xffffffffu, live[0] && first[0]), lead1 = __ballot_sync(0xffffffffu, live[1] && first[1]);
  const int nR = __popc(lead0) + __popc(lead1);
  int slot[2] = {-1, -1}, ent[2] = {0, 0};
  bool ok = nR <= a.C;
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    if (live[h] && first[h]) {
      slot[h] = sh.pi[e[h]];
      ok = ok && slot[h] >= 0;
    }
  }
  if (!__all_sync(0xffffffffu, ok)) return false;
  // position of every first-pair among the first-pairs in sorted order: pairs are scattered by pos through shared scratch
  if (lane < 2) sh.bitmap[lane] = 0u;
  __syncwarp();
#pragma unroll
  for (int h = 0; h < 2; ++h)
    if (live[h] && first[h]) atomicOr(&sh.bitmap[pos[h] >> 5], 1u << (pos[h] & 31));
  __syncwarp();
  const unsigned b0 = sh.bitmap[0], b1 = sh.bitmap[1];
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    if (!live[h]) continue;
    const int p = lane + 32 * h;
    a.plan.pair_list[pos[h]] = p;
    if (a.plan.pair_pos) a.plan.pair_pos[p] = pos[h];
    if (!first[h]) continue;
    ent[h] = pos[h] < 32 ? __popc(b0 & ((1u << pos[h]) - 1u)) : __popc(b0) + __popc(b1 & ((1u << (pos[h] - 32)) - 1u));
    const int i = ent[h];
    a.plan.entry_expert[i] = e[h]; a.plan.entry_slot[i] = slot[h]; a.plan.entry_miss[i] = 0;
    a.plan.exp_count[e[h]] = cnt[h]; a.plan.exp_offset[e[h]] = pos[h];
    if (a.plan.unit_entry) a.plan.unit_entry[i] = i;
    if (writer) {                                                  // line 9: the tick
      a.st.tau[slot[h]] = sh.clock + 1ull;
      a.st.freq[e[h]] = sh.freq[e[h]] + 1ull;
      if (a.trace_on) {
        const u64 base = a.trace_ctr[0];
        if (base + (u64)nR <= a.trace_cap) {
          wisp_trace_event ev;
          ev.step = sh.scal[1]; ev.layer = (uint32_t)a.layer; ev.wave = 0u; ev.expert = e[h]; ev.slot = slot[h]; ev.evicted = -1; ev.kind = 0u;
          a.trace[base + i] = ev;
        }
      }
    }
  }
  __syncwarp();
  if (lane == 0) {
    a.plan.hdr[0] = nR > 0 ? 1 : 0; a.plan.hdr[1] = nR; a.plan.hdr[2] = 0; a.plan.hdr[3] = n_pairs;
    a.plan.exp_offset[E] = n_pairs;
    if (writer) {
      a.st.scal[0] = sh.clock + 1ull;
      if (nR > 0) a.st.scal[1] = sh.scal[1] + 1ull;
      a.st.scal[2] = sh.scal[2] + (u64)nR;
      a.st.scal[5] = sh.scal[5] + (u64)nR;
      if (a.trace_on) {
        const u64 base = a.trace_ctr[0];
        if (base + (u64)nR <= a.trace_cap) a.trace_ctr[0] = base + (u64)nR;
        else a.trace_ctr[1] += (u64)nR;
      }
    }
  }
  __syncwarp();
  return true;
}

__global__ void __launch_bounds__(kPlanThreads) residency_plan_kernel(PlanArgs a) {
  __shared__ PlanShared<kPlanThreads> sh;
  plan_load<kPlanThreads>(sh, a.st, a.E, a.C);
  __syncthreads();
  plan_compute<kPlanThreads>(a, sh, /*writer=*/true, /*bar=*/0);
}

// Stable grouping of (token, rank) pairs by expert for large n_pairs: one CTA of kGroupThreads per expert, ONE pass: thread t
// owns the contiguous range of pairs [t * per, (t + 1) * per), counts its matches, an exclusive block scan of the counts gives
// the position of its first match, and it writes its matches in ascending pair order (so the order inside an expert is ascending).
constexpr int kGroupThreads = 1024;
__global__ void __launch_bounds__(kGroupThreads) group_pairs_kernel(const int* __restrict__ ids, int n_pairs, PlanPtrs plan) {
  constexpr int NW = kGroupThreads / 32;
  __shared__ int s_ws[NW];
  const int e = blockIdx.x;
  if (plan.exp_count[e] == 0) return;
  const int pos0 = plan.exp_offset[e];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int per = (((n_pairs + kGroupThreads - 1) / kGroupThreads) + 3) & ~3;      // multiple of 4: int4 loads
  const int lo = min(n_pairs, (int)threadIdx.x * per), hi = min(n_pairs, lo + per);
  const bool vec = (n_pairs & 3) == 0;
  int cnt = 0;
  if (vec) {
    for (int p = lo; p < hi; p += 4) {
      const int4 v = __ldg(reinterpret_cast<const int4*>(ids + p));
      cnt += (v.x == e) + (v.y == e) + (v.z == e) + (v.w == e);
    }
  } else {
    for (int p = lo; p < hi; ++p) cnt += ids[p] == e;
  }
  int inc = cnt;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += v; }
  if (lane == 31) s_ws[wid] = inc;
  __syncthreads();
  int before = inc - cnt;
  for (int i = 0; i < wid; ++i) before += s_ws[i];
  if (cnt == 0) return;
  int pos = pos0 + before;
  for (int p = lo; p < hi; ++p)
    if (ids[p] == e) plan.pair_list[pos++] = p;
}

// ---- resize (a7, G13) -------------------------------------------------------
// One CTA, one layer.  Shrink: keep the C_new best residents (LRU: tau desc, slot asc; LFU: f desc, tau
// desc, slot asc), drop the rest, move survivors living in slots >= C_new to the lowest free slots.
// moves[2*i] = src slot, moves[2*i+1] = dst slot; *n_moves = count.  Grow: new slots empty, tau = 0.
struct ResizeArgs {
  int E, C_old, C_new, policy, layer;
  LayerState st;
  int* moves;
  int* n_moves;
  wisp_trace_event* trace;
  u64* trace_ctr;
  u64 trace_cap;
  int trace_on;
};

__global__ void __launch_bounds__(kPlanThreads) residency_resize_kernel(ResizeArgs a) {
  __shared__ int s_pinv[kMaxExperts];
  __shared__ u64 s_tau[kMaxExperts];
  __shared__ u64 s_f[kMaxExperts];
  __shared__ unsigned char s_keep[kMaxExperts];
  __shared__ int s_ws[33];
  const int tid = threadIdx.x;
  const int Co = a.C_old, Cn = a.C_new;
  if (Cn >= Co) {
    if (tid >= Co && tid < Cn) { a.st.pi_inv[tid] = -1; a.st.tau[tid] = 0; }
    if (tid == 0) *a.n_moves = 0;
    return;
  }
  if (tid < Co) {
    s_pinv[tid] = a.st.pi_inv[tid];
    s_tau[tid] = a.st.tau[tid];
    s_f[tid] = (a.policy == WISP_LFU && s_pinv[tid] >= 0) ? a.st.freq[s_pinv[tid]] : 0ull;
  }
  __syncthreads();
  int occ = -1, keep = 0;
  if (tid < Co) {
    occ = s_pinv[tid];
    if (occ >= 0) {
      int rank = 0;   // number of occupied slots that come before this one in the keep order
      for (int o = 0; o < Co; ++o) {
        if (o == tid || s_pinv[o] < 0) continue;
        bool before;
        if (s_f[o] != s_f[tid]) before = s_f[o] > s_f[tid];
        else if (s_tau[o] != s_tau[tid]) before = s_tau[o] > s_tau[tid];
        else before = o < tid;
        rank += before;
      }
      keep = rank < Cn;
    }
    s_keep[tid] = (unsigned char)keep;
  }
  __syncthreads();
  const int is_drop = (tid < Co && occ >= 0 && !keep);
  const int is_move = (tid < Co && keep && tid >= Cn);
  const int is_free = (tid < Cn && !(occ >= 0 && keep));
  int n_drop, n_move, n_free;
  const int di = block_excl_scan<kPlanThreads>(is_drop, s_ws, n_drop, 0);
  const int mi = block_excl_scan<kPlanThreads>(is_move, s_ws, n_move, 0);
  const int fi = block_excl_scan<kPlanThreads>(is_free, s_ws, n_free, 0);
  __shared__ int s_free[kMaxExperts];
  if (is_free) s_free[fi] = tid;
  __syncthreads();
  bool trace_ok = false;
  u64 tb = 0;
  if (a.trace_on) { tb = a.trace_ctr[0]; trace_ok = tb + (u64)(n_drop + n_move) <= a.trace_cap; }
  const u64 step_no = a.st.scal[1];
  if (is_drop) {
    a.st.pi[occ] = -1;
    a.st.pi_inv[tid] = -1;
    a.st.tau[tid] = 0;
    if (trace_ok) {
      wisp_trace_event ev;
      ev.step = step_no; ev.layer = (uint32_t)a.layer; ev.wave = 0; ev.expert = occ; ev.slot = tid; ev.evicted = -1; ev.kind = 2u;
      a.trace[tb + di] = ev;
    }
  }
  __syncthreads();
  if (is_move) {
    const int dst = s_free[mi];
    a.st.pi[occ] = dst;
    a.st.pi_inv[dst] = occ;
    a.st.tau[dst] = s_tau[tid];
    a.st.pi_inv[tid] = -1;
    a.st.tau[tid] = 0;
    a.moves[2 * mi] = tid;
    a.moves[2 * mi + 1] = dst;
    if (trace_ok) {
      wisp_trace_event ev;
      ev.step = step_no; ev.layer = (uint32_t)a.layer; ev.wave = 0; ev.expert = occ; ev.slot = dst; ev.evicted = tid; ev.kind = 3u;
      a.trace[tb + n_drop + mi] = ev;
    }
  }
  if (tid == 0) {
    *a.n_moves = n_move;
    if (a.trace_on) {
      if (trace_ok) a.trace_ctr[0] = tb + (u64)(n_drop + n_move);
      else a.trace_ctr[1] += (u64)(n_drop + n_move);
    }
  }
}

}  // namespace wisp

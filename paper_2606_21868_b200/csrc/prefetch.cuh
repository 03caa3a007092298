// prefetch.cuh -- SURVEY.md 8(f) f3: the online co-activation predictor of App. E and the speculative
// expert prefetch whose failure is the paper's central finding (Section 4: "speculative copies compete with
// demand copies for the same link, and at tight caps they can evict experts that the next step still needs").
//
//   A_{l,l'}(e,e')   co-activation counts, P_{l,l'}(e'|e) = A / sum_j A(e,j), s_{l'}(e') = sum_{l<l'} gamma^{l'-l} sum_{e in R_l} P(e'|e)
//
// Built for the split decode form only (WISP_FETCH_ZEROCOPY): after layer l's plan, ONE CTA (predict_prefetch_kernel)
//   1. adds this forward pass to the tables whose target is layer l (sources: the `window` layers before it);
//   2. scores every expert of layer l+1 from the layers routed so far -- fp64, explicit round-to-nearest operations in the
//      order fixed in oracle/predictor.py, so the ranking is bit-identical to the oracle's;
//   3. takes the n best-scoring experts that are absent and have a positive score (score desc, id asc), gives each the next
//      victim slot of layer l+1 in increasing policy key (tau <- clock, no tick; G27), emits trace events of kind 4
//      and a copy list;
// and a copy kernel on the SIDE stream streams them from the mapped master while layer l's FFN runs on the main stream.
// Layer l+1 waits for the copies before its own demand fetch.  Outputs never depend on any of this.
#pragma once
#include "common.cuh"
#include "residency.cuh"

namespace wisp {

constexpr int kPredictThreads = 256;
constexpr int kMaxPrefetch = 32;          // experts prefetched per layer call
constexpr int kMaxWindow = 4;             // source layers per target

struct PredictArgs {
  int L, E, C, policy, layer;             // layer = l, the layer that has just routed; the prefetch target is l + 1
  int window, n_prefetch;
  double gpow[kMaxWindow + 1];            // gamma^dist as running products (host, fp64)
  const int* entry_expert;                // plan of layer l (global): its routed set R_l
  const int* plan_hdr;
  unsigned* A;                            // [L][window][E][E] counts, target-major
  unsigned* row;                          // [L][window][E] source marginals
  int* rlist;                             // [L][E] ascending routed ids of the pass in progress
  int* rcount;                            // [L]
  LayerState st_next;                     // residency state of layer l + 1
  int* copy_list;                         // [0] = count, then (expert, slot) pairs
  wisp_trace_event* trace;
  u64* trace_ctr;
  u64 trace_cap;
  int trace_on;
};

__global__ void __launch_bounds__(kPredictThreads) predict_prefetch_kernel(PredictArgs a) {
  __shared__ unsigned s_bits[kMaxExperts / 32];
  __shared__ int s_R[kMaxWindow + 1][256];           // routed lists: [0] = layer l, [d] = layer l - d  (|R| <= 256 in decode)
  __shared__ int s_nR[kMaxWindow + 1];
  __shared__ double s_score[kMaxExperts];
  __shared__ unsigned char s_elig[kMaxExperts];
  __shared__ int s_pick[kMaxPrefetch], s_victim[kMaxPrefetch];
  __shared__ int s_npick;
  const int tid = threadIdx.x, E = a.E, l = a.layer;
  const size_t EE = (size_t)E * E;

  // ---- R_l, ascending: bitmap of the plan's entries, then enumerate ----
  for (int i = tid; i < kMaxExperts / 32; i += kPredictThreads) s_bits[i] = 0u;
  if (tid == 0) s_npick = 0;
  __syncthreads();
  const int nR = a.plan_hdr[1];
  for (int i = tid; i < nR; i += kPredictThreads) { const int e = a.entry_expert[i]; atomicOr(&s_bits[e >> 5], 1u << (e & 31)); }
  __syncthreads();
  if (tid == 0) {
    int n = 0;
    for (int w = 0; w < (E + 31) / 32; ++w) {
      unsigned bits = s_bits[w];
      while (bits) { const int b = __ffs(bits) - 1; bits &= bits - 1; if (n < 256) s_R[0][n] = w * 32 + b; ++n; }
    }
    s_nR[0] = min(n, 256);
    a.rcount[l] = s_nR[0];
  }
  __syncthreads();
  for (int i = tid; i < s_nR[0]; i += kPredictThreads) a.rlist[(size_t)l * E + i] = s_R[0][i];
  for (int dist = 1; dist <= a.window; ++dist) {
    const int src = l - dist;
    if (tid == 0) s_nR[dist] = src >= 0 ? min(a.rcount[src], 256) : 0;
    __syncthreads();
    for (int i = tid; i < s_nR[dist]; i += kPredictThreads) s_R[dist][i] = a.rlist[(size_t)src * E + i];
  }
  __syncthreads();

  // ---- 1. this pass enters the tables whose TARGET is layer l ----
  for (int dist = 1; dist <= a.window; ++dist) {
    const int ns = s_nR[dist], nt = s_nR[0];
    unsigned* A = a.A + ((size_t)l * a.window + (dist - 1)) * EE;
    unsigned* row = a.row + ((size_t)l * a.window + (dist - 1)) * E;
    for (int i = tid; i < ns * nt; i += kPredictThreads) A[(size_t)s_R[dist][i / nt] * E + s_R[0][i % nt]] += 1u;   // distinct cells
    for (int i = tid; i < ns; i += kPredictThreads) row[s_R[dist][i]] += (unsigned)nt;
  }
  if (l + 1 >= a.L || a.n_prefetch <= 0) { if (tid == 0) a.copy_list[0] = 0; return; }
  __syncthreads();

  // ---- 2. scores of the experts of layer l + 1: nearest source first, source experts ascending (oracle/predictor.py) ----
  const int target = l + 1;
  for (int e2 = tid; e2 < E; e2 += kPredictThreads) {
    double s = 0.0;
    for (int dist = 1; dist <= a.window; ++dist) {
      const int src = target - dist;                    // = l - (dist - 1): the list s_R[dist - 1]
      if (src < 0) continue;
      const unsigned* A = a.A + ((size_t)target * a.window + (dist - 1)) * EE;
      const unsigned* row = a.row + ((size_t)target * a.window + (dist - 1)) * E;
      const double g = a.gpow[dist];
      for (int i = 0; i < s_nR[dist - 1]; ++i) {
        const int e = s_R[dist - 1][i];
        const unsigned r = row[e];
        if (r == 0u) continue;
        s = __dadd_rn(s, __dmul_rn(__ddiv_rn((double)A[(size_t)e * E + e2], (double)r), g));
      }
    }
    s_score[e2] = s;
    s_elig[e2] = (s > 0.0 && a.st_next.pi[e2] < 0) ? 1 : 0;
  }
  __syncthreads();
  // ---- 3. the n best eligible candidates (score desc, id asc) by rank counting ----
  const int n_want = min(min(a.n_prefetch, kMaxPrefetch), a.C);
  for (int e2 = tid; e2 < E; e2 += kPredictThreads) {
    if (!s_elig[e2]) continue;
    const double s = s_score[e2];
    int rank = 0;
    for (int o = 0; o < E; ++o)
      if (s_elig[o] && (s_score[o] > s || (s_score[o] == s && o < e2))) ++rank;
    if (rank < n_want) { s_pick[rank] = e2; atomicAdd(&s_npick, 1); }
  }
  __syncthreads();
  const int np = s_npick;                                 // ranks 0..np-1 are all filled (ranks are a permutation of the eligible set)
  // victims of layer l + 1: all slots in increasing policy key; the i-th pick takes the i-th victim
  for (int sl = tid; sl < a.C; sl += kPredictThreads) {
    const int occ = a.st_next.pi_inv[sl];
    const u64 kf = a.policy == WISP_LFU ? (occ < 0 ? 0ull : a.st_next.freq[occ] + 1ull) : 0ull, kt = a.st_next.tau[sl];
    int rank = 0;
    for (int o = 0; o < a.C; ++o) {
      const int oo = a.st_next.pi_inv[o];
      const u64 of = a.policy == WISP_LFU ? (oo < 0 ? 0ull : a.st_next.freq[oo] + 1ull) : 0ull;
      if (key_less(of, a.st_next.tau[o], o, kf, kt, sl)) ++rank;
    }
    if (rank < np) s_victim[rank] = sl;
  }
  __syncthreads();
  if (tid == 0) {
    const u64 clock = a.st_next.scal[0], step_no = a.st_next.scal[1];
    bool trace_ok = false;
    u64 tb = 0;
    if (a.trace_on) { tb = a.trace_ctr[0]; trace_ok = tb + (u64)np <= a.trace_cap; }
    int evict = 0;
    for (int i = 0; i < np; ++i) {
      const int e = s_pick[i], sl = s_victim[i], old = a.st_next.pi_inv[sl];
      if (old >= 0) { a.st_next.pi[old] = -1; ++evict; }
      a.st_next.pi[e] = sl;
      a.st_next.pi_inv[sl] = e;
      a.st_next.tau[sl] = clock;
      a.copy_list[1 + 2 * i] = e;
      a.copy_list[2 + 2 * i] = sl;
      if (trace_ok) {
        wisp_trace_event ev;
        ev.step = step_no; ev.layer = (uint32_t)target; ev.wave = 0u; ev.expert = e; ev.slot = sl; ev.evicted = old; ev.kind = 4u;
        a.trace[tb + i] = ev;
      }
    }
    a.copy_list[0] = np;
    a.st_next.scal[4] += (u64)evict;
    a.st_next.scal[7] += (u64)np;                         // prefetches of this layer
    if (a.trace_on) {
      if (trace_ok) a.trace_ctr[0] = tb + (u64)np;
      else a.trace_ctr[1] += (u64)np;
    }
  }
}

// Copies the experts of a copy list from the mapped master of `layer` into their slots (zero-copy reads over the host link).
__global__ void __launch_bounds__(256) prefetch_copy_kernel(const int* __restrict__ copy_list, const uint4* __restrict__ master,
                                                           uint4* __restrict__ pool, size_t blob_vec, int L, int layer) {
  const int n = copy_list[0];
  for (int i = 0; i < n; ++i) {
    const uint4* src = master + (size_t)copy_list[1 + 2 * i] * blob_vec;
    uint4* dst = pool + ((size_t)copy_list[2 + 2 * i] * L + layer) * blob_vec;
    for (size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v < blob_vec; v += (size_t)gridDim.x * blockDim.x) dst[v] = __ldcs(src + v);
  }
}

}  // namespace wisp

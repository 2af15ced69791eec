// Plan kernels of the ForeMoE hot path (sm_100a): load histogram (a1), Stage-4 integer quotas
// (a2), replica assignment + stable counting-sort destinations (a3/a4).
// Contract: include/foremoe.h.  Rule and readings: DESIGN.md sec. 3.
#include <limits.h>

#include "foremoe_data.cuh"

namespace foremoe {

// =============================================================================================
// a1: load histogram  (w_{s,e}, PAPER.md:204 / :247, single source rank)
//
// Tiles are fixed token ranges of one layer; a tile may straddle micro-step boundaries, so it is
// walked segment by segment, each segment counted into a shared-memory histogram and flushed to
// hist[i][l][:] with one global atomic per non-zero bin.
// kMode 0: one shared atomic per pair, 4-byte coalesced loads.
// kMode 1: warp-aggregated: lanes holding the same expert id elect a leader that adds the group's
//          population once (match.any) -- one shared atomic per distinct id and warp.
// kMode 2: one shared atomic per pair, 16-byte loads (4 pairs per lane), 4 loads in flight (default:
//          fastest on every config incl. the all-one-expert worst case, profiles/r01_hist.md).
// =============================================================================================
// Count the ids src[0..n) into the shared-memory histogram sh[E]: one shared atomic per pair,
// 16-byte loads (head / tail handled 4 bytes at a time), 4 loads in flight per thread.
// Returns FOREMOE_FAULT_ID_RANGE if an id outside [0, E) was seen (it is not counted).
__device__ __forceinline__ int count_ids(const int32_t *__restrict__ src, int n, int32_t *sh, int E) {
  int fault = 0;
  auto count = [&](int e) {
    if ((unsigned)e < (unsigned)E) atomicAdd(&sh[e], 1); else fault = FOREMOE_FAULT_ID_RANGE;
  };
  const int tid = threadIdx.x, nt = blockDim.x;
  int head = (int)(((16 - ((uintptr_t)src & 15)) & 15) >> 2);
  if (head > n) head = n;
  if (tid < head) count(__ldg(src + tid));
  const int4 *v4 = (const int4 *)(src + head);
  const int nv = (n - head) >> 2;
  int v = tid;
  for (; v + 3 * nt < nv; v += 4 * nt) {
    const int4 a = __ldg(v4 + v), b = __ldg(v4 + v + nt);
    const int4 c = __ldg(v4 + v + 2 * nt), d = __ldg(v4 + v + 3 * nt);
    count(a.x); count(a.y); count(a.z); count(a.w);
    count(b.x); count(b.y); count(b.z); count(b.w);
    count(c.x); count(c.y); count(c.z); count(c.w);
    count(d.x); count(d.y); count(d.z); count(d.w);
  }
  for (; v < nv; v += nt) {
    const int4 a = __ldg(v4 + v);
    count(a.x); count(a.y); count(a.z); count(a.w);
  }
  const int done = head + (nv << 2);
  if (tid < n - done) count(__ldg(src + done + tid));
  return fault;
}

template <int kMode>
__global__ void __launch_bounds__(256)
k_load_hist(const int32_t *__restrict__ ids, const int32_t *__restrict__ mb_off, int L, int T, int K,
            int E, int n_mb, int tile_tokens, int tiles_per_layer, int32_t *__restrict__ hist,
            int32_t *dev_status) {
  extern __shared__ int32_t sh[];   // [E]
  const int tid = threadIdx.x;
  const int lane = tid & 31;

  // every CTA validates the boundaries itself (n_mb + 1 ints): no workspace in this entry point
  int bad = 0;
  for (int i = tid; i <= n_mb; i += blockDim.x) {
    int v = mb_off[i];
    if (i == 0 && v != 0) bad = 1;
    if (i == n_mb && v != T) bad = 1;
    if (i < n_mb && mb_off[i + 1] < v) bad = 1;
  }
  bad = __syncthreads_or(bad);
  if (bad) {
    if (blockIdx.x == 0 && tid == 0) raise_fault(dev_status, FOREMOE_FAULT_MB_OFF);
    return;
  }

  int fault = 0;
  const int n_tiles = L * tiles_per_layer;
  for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const int l = tile / tiles_per_layer;
    int t0 = (tile - l * tiles_per_layer) * tile_tokens;
    const int t1 = min(T, t0 + tile_tokens);
    if (t0 >= t1) continue;
    int i = find_range(mb_off, n_mb, t0);
    const int32_t *lids = ids + (size_t)l * T * K;
    while (t0 < t1) {
      const int seg_end = min(t1, __ldg(mb_off + i + 1));
      for (int e = tid; e < E; e += blockDim.x) sh[e] = 0;
      __syncthreads();
      const int p0 = t0 * K, p1 = seg_end * K;
      if (kMode == 2) {
        fault |= count_ids(lids + p0, p1 - p0, sh, E);
      } else {
        // uniform trip count so that every lane takes part in match.any
        for (int p = p0 + tid - lane; p < p1; p += blockDim.x) {
          const int pp = p + lane;
          int e = pp < p1 ? __ldg(lids + pp) : -1;
          const bool ok = (unsigned)e < (unsigned)E;
          if (pp < p1 && !ok) fault = FOREMOE_FAULT_ID_RANGE;
          if (kMode == 1) {
            const unsigned key = ok ? (unsigned)e : (0x80000000u | lane);
            const unsigned grp = __match_any_sync(0xffffffffu, key);
            if (ok && lane == __ffs(grp) - 1) atomicAdd(&sh[e], __popc(grp));
          } else {
            if (ok) atomicAdd(&sh[e], 1);
          }
        }
      }
      __syncthreads();
      int32_t *dst = hist + ((size_t)i * L + l) * E;
      for (int e = tid; e < E; e += blockDim.x) {
        const int v = sh[e];
        if (v) atomicAdd(dst + e, v);
      }
      __syncthreads();
      t0 = seg_end;
      ++i;
      while (i < n_mb && __ldg(mb_off + i + 1) <= t0) ++i;   // skip empty micro-steps
    }
  }
  if (fault) raise_fault(dev_status, fault);
}

// step aggregate  w-bar_{s,e} = sum_i w^{(i)}_{s,e}
__global__ void k_step_hist(const int32_t *__restrict__ hist, int n_mb, int LE,
                            int64_t *__restrict__ step_hist) {
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  if (x >= LE) return;
  int64_t s = 0;
  for (int i = 0; i < n_mb; i++) s += hist[(size_t)i * LE + x];
  step_hist[x] = s;
}

// =============================================================================================
// assign, step 0: micro-step tables.  chunk_off[i] = number of ranking chunks before micro-step i
// (a chunk = up to tpc consecutive tokens of ONE instance).  One CTA.
// =============================================================================================
__global__ void k_mb_tables(const int32_t *__restrict__ mb_off, int n_mb, int T, int tpc,
                            int32_t *__restrict__ chunk_off, int32_t *__restrict__ mb_ok,
                            int32_t *dev_status) {
  int bad = 0;
  for (int i = threadIdx.x; i <= n_mb; i += blockDim.x) {
    int v = mb_off[i];
    if (i == 0 && v != 0) bad = 1;
    if (i == n_mb && v != T) bad = 1;
    if (i < n_mb && mb_off[i + 1] < v) bad = 1;
  }
  bad = __syncthreads_or(bad);
  if (threadIdx.x == 0) {
    *mb_ok = !bad;
    int run = 0;
    for (int i = 0; i < n_mb; i++) {
      chunk_off[i] = run;
      if (!bad) run += (mb_off[i + 1] - mb_off[i] + tpc - 1) / tpc;
    }
    chunk_off[n_mb] = run;
    if (bad) raise_fault(dev_status, FOREMOE_FAULT_MB_OFF);
  }
}

// =============================================================================================
// assign, step 1: per-placement tables.  One CTA per placement (layer, or (micro-step, layer)).
//   host_ptr/host_slot : CSR list of ALL slots holding expert e, ascending slot index
//   active[j]          : slot j is the lowest-indexed slot of its expert on its rank (reading 10)
//   rslot[r*Ns + s]    : active slots of rank r ordered by ascending expert id, then -1 padding
// =============================================================================================
__global__ void __launch_bounds__(256)
k_placement_tables(const int32_t *__restrict__ slot_expert, int E, int S, int Ns, int P,
                   int32_t *__restrict__ host_ptr, int32_t *__restrict__ host_slot,
                   int32_t *__restrict__ active, int32_t *__restrict__ rslot,
                   int32_t *__restrict__ pl_fault, int32_t *dev_status) {
  extern __shared__ int32_t sm[];
  int32_t *se = sm;            // [S]
  int32_t *cnt = sm + S;       // [E+1]
  int32_t *act = cnt + E + 1;  // [S]
  const int pl = blockIdx.x;
  const int32_t *src = slot_expert + (size_t)pl * S;
  host_ptr += (size_t)pl * (E + 1);
  host_slot += (size_t)pl * S;
  active += (size_t)pl * S;
  rslot += (size_t)pl * S;

  int bad = 0;
  for (int j = threadIdx.x; j < S; j += blockDim.x) {
    int e = src[j];
    if (e < -1 || e >= E) { bad = 1; e = -1; }
    se[j] = e;
  }
  bad = __syncthreads_or(bad);
  for (int e = threadIdx.x; e <= E; e += blockDim.x) cnt[e] = 0;
  __syncthreads();
  for (int j = threadIdx.x; j < S; j += blockDim.x) {
    const int e = se[j];
    if (e >= 0) atomicAdd(&cnt[e], 1);
    int a = e >= 0;
    for (int j2 = (j / Ns) * Ns; j2 < j; j2++) a &= (se[j2] != e);
    act[j] = a;
    active[j] = a;
  }
  __syncthreads();
  {   // exclusive prefix of cnt[0..E): every thread scans a contiguous run, thread 0 the run totals
    __shared__ int part[256];
    const int per = (E + blockDim.x - 1) / blockDim.x;
    const int e0 = min(E, (int)threadIdx.x * per), e1 = min(E, e0 + per);
    int sum = 0;
    for (int e = e0; e < e1; e++) sum += cnt[e];
    part[threadIdx.x] = sum;
    __syncthreads();
    if (threadIdx.x == 0) {
      int run = 0;
      for (int t = 0; t < (int)blockDim.x; t++) { const int n = part[t]; part[t] = run; run += n; }
      cnt[E] = run;
      pl_fault[pl] = bad;
      if (bad) raise_fault(dev_status, FOREMOE_FAULT_SLOT_EXPERT);
    }
    __syncthreads();
    int run = part[threadIdx.x];
    for (int e = e0; e < e1; e++) { const int n = cnt[e]; cnt[e] = run; run += n; }
  }
  __syncthreads();
  for (int e = threadIdx.x; e <= E; e += blockDim.x) host_ptr[e] = cnt[e];
  __syncthreads();
  // host list of every expert in ascending slot index: slots claim a position of their expert's
  // segment in any order, then every (short) segment is sorted
  for (int j = threadIdx.x; j < S; j += blockDim.x) {
    const int e = se[j];
    if (e >= 0) host_slot[atomicAdd(&cnt[e], 1)] = j;
  }
  __syncthreads();
  for (int e = threadIdx.x; e < E; e += blockDim.x) {
    const int a0 = host_ptr[e], a1 = cnt[e];               // cnt[e] has advanced to the segment's end
    for (int a = a0 + 1; a < a1; a++) {
      const int v = host_slot[a];
      int b = a - 1;
      for (; b >= a0 && host_slot[b] > v; b--) host_slot[b + 1] = host_slot[b];
      host_slot[b + 1] = v;
    }
  }
  // active slots of each rank by ascending expert id (they hold distinct experts)
  for (int j = threadIdx.x; j < S; j += blockDim.x) {
    const int r0 = (j / Ns) * Ns;
    if (act[j]) {
      int pos = 0;
      for (int j2 = r0; j2 < r0 + Ns; j2++) pos += (act[j2] && se[j2] < se[j]);
      rslot[r0 + pos] = j;
    }
    int n_act = 0;
    for (int j2 = r0; j2 < r0 + Ns; j2++) n_act += act[j2];
    if (j - r0 >= n_act) rslot[j] = -1;
  }
}

// =============================================================================================
// assign, step 2: per-chunk expert counts (input of the stable ranking).
// grid (max_chunks, L).
// =============================================================================================
struct ChunkInfo { int i, t0, t1; };

__device__ __forceinline__ bool locate_chunk(const int32_t *__restrict__ chunk_off,
                                             const int32_t *__restrict__ mb_off, int n_mb, int tpc,
                                             int c, ChunkInfo *ci) {
  if (c >= __ldg(chunk_off + n_mb)) return false;
  const int i = find_range(chunk_off, n_mb, c);
  ci->i = i;
  ci->t0 = __ldg(mb_off + i) + (c - __ldg(chunk_off + i)) * tpc;
  ci->t1 = min(__ldg(mb_off + i + 1), ci->t0 + tpc);
  return true;
}

__global__ void __launch_bounds__(kChunkThreads)
k_chunk_hist(const int32_t *__restrict__ ids, const int32_t *__restrict__ mb_off,
             const int32_t *__restrict__ chunk_off, int L, int T, int K, int E, int n_mb, int tpc,
             int max_chunks, int32_t *__restrict__ chunk_cnt, int32_t *__restrict__ hist_out,
             int32_t *dev_status) {
  extern __shared__ int32_t sh[];   // [E]
  ChunkInfo ci;
  const int c = blockIdx.x, l = blockIdx.y;
  if (!locate_chunk(chunk_off, mb_off, n_mb, tpc, c, &ci)) return;
  for (int e = threadIdx.x; e < E; e += blockDim.x) sh[e] = 0;
  __syncthreads();
  // hist_out / dev_status are non-NULL only in foremoe_plan, where this pass also stands in for
  // k_load_hist: a chunk lies inside one instance, so hist[i][l][:] is the sum of its chunks' counts
  const int fault = count_ids(ids + ((size_t)l * T + ci.t0) * K, (ci.t1 - ci.t0) * K, sh, E);
  if (fault) raise_fault(dev_status, fault);
  __syncthreads();
  int32_t *dst = chunk_cnt + ((size_t)l * max_chunks + c) * E;
  int32_t *hdst = hist_out ? hist_out + ((size_t)ci.i * L + l) * E : nullptr;
  for (int e = threadIdx.x; e < E; e += blockDim.x) {
    const int v = sh[e];
    dst[e] = v;
    if (hdst && v) atomicAdd(hdst + e, v);
  }
}

// =============================================================================================
// assign, step 3: one CTA per instance.
//   warp 0   : Stage-4 integer quotas by the exact water-filling rule (O2):
//              Phase A forced loads, Phase B Gauss-Seidel water-filling passes to a fixpoint
//              ("assign each token unit to the replica whose rank has the
//              smallest accumulated load", :844-846), Phase C unit augmentations.
//   warps 1+ : exclusive scan of the instance's chunk counts over chunks (per expert).
// then quota / rank_load / slot_off and the pair-lookup tables are written by all threads.
// =============================================================================================
// Index-valued tables (slots, experts, ranks, small counts) are held as I = int32_t, or int16_t when
// E and S stay below 2^15 and the 32-bit layout would let shared memory cap the resident CTAs: the
// commodity instances of the per-source plan (E * M, S * M) are large, one warp per instance does the
// sequential work, and the kernel's rate is the number of instances resident per SM.
template <typename I>
struct QuotaSmemT {
  int32_t *c, *q, *load, *visited, *par_rank, *par_from, *par_to, *queue, *soff;
  I *se, *hptr, *ahs, *rk, *rslot, *R, *nact;
  // Phase B bookkeeping: stamp[r] = event number of the last change of load[r]; seen[e] = event
  // number at e's last fill.  A fill is a pure function of its hosts' loads (own quota removed) and
  // c[e], so when no host rank was touched since e's last fill it would reproduce the same quotas:
  // it is skipped.  The result is unchanged bit for bit; late passes cost almost nothing.
  int32_t *stamp, *seen;
};
// hptr: CSR offsets of the slots of expert e; ahs[hptr[e] .. hptr[e] + nact[e]): its ACTIVE host
// slots (ascending); rk[j] = rank of slot j.

// One replicated expert: closed form of the unit-by-unit fill.  With host loads l_j (the expert's
// own quota removed), lam = largest integer with sum_j max(0, lam - l_j) <= c; every host gets
// max(0, lam - l_j); the remaining units go one each to the first hosts (ascending slot index)
// among {l_j <= lam}.  Serial version (one lane), used when an expert has more than 32 hosts.
template <typename I>
__device__ __forceinline__ int water_fill_expert(const QuotaSmemT<I> &s, int e) {
  const int a0 = s.hptr[e], a1 = a0 + s.nact[e];
  int cur = INT_MAX;
  for (int a = a0; a < a1; a++) {
    const int j = s.ahs[a], r = s.rk[j];
    const int lj = s.load[r] - s.q[j];
    s.load[r] = lj;
    cur = min(cur, lj);
  }
  int64_t rem = s.c[e];
  int lam;
  for (;;) {
    int m = 0, nxt = INT_MAX;
    for (int a = a0; a < a1; a++) {
      const int lj = s.load[s.rk[s.ahs[a]]];
      if (lj <= cur) m++; else nxt = min(nxt, lj);
    }
    if (nxt == INT_MAX || rem < (int64_t)(nxt - cur) * m) {
      lam = cur + (int)(rem / m);
      rem = rem % m;
      break;
    }
    rem -= (int64_t)(nxt - cur) * m;
    cur = nxt;
  }
  int changed = 0;
  for (int a = a0; a < a1; a++) {
    const int j = s.ahs[a], r = s.rk[j];
    const int lj = s.load[r];
    int g = 0;
    if (lj <= lam) {
      g = lam - lj;
      if (rem > 0) { g++; rem--; }
    }
    changed |= (g != s.q[j]);
    s.q[j] = g;
    s.load[r] = lj + g;
  }
  return changed;
}

// Warp version of the same closed form (all 32 lanes call it; lane a owns the a-th active host).
// f_a = sum_b max(0, l_a - l_b) is what it costs to raise every lower host to l_a; the water level
// sits on top of the highest host load l* with f(l*) <= c:  lam = l* + (c - f(l*)) / m,
// m = #{l_b <= l*}, and (c - f(l*)) % m units are left for the lowest slots among those m hosts.
template <typename I>
__device__ __forceinline__ int water_fill_expert_warp(const QuotaSmemT<I> &s, int e, int lane, int &event) {
  const unsigned full = 0xffffffffu;
  const int a0 = s.hptr[e], h = s.nact[e];
  if (h > 32) {
    int ch = 0;
    if (lane == 0) ch = water_fill_expert(s, e);
    __syncwarp();
    ch = __shfl_sync(full, ch, 0);
    if (ch) {                                    // conservative: every host rank counts as touched
      event++;
      for (int a = a0 + lane; a < a0 + h; a += 32) s.stamp[s.rk[s.ahs[a]]] = event;
      __syncwarp();
    }
    return ch;
  }
  const bool on = lane < h;
  int j = 0, r = 0, qold = 0, l = INT_MAX;
  if (on) { j = s.ahs[a0 + lane]; r = s.rk[j]; }
  if (__reduce_max_sync(full, on ? s.stamp[r] : 0) <= s.seen[e]) return 0;   // hosts untouched: same result
  if (on) { qold = s.q[j]; l = s.load[r] - qold; }
  const int c = s.c[e];
  long long f = 0;
  for (int b = 0; b < h; b++) {
    const int lb = __shfl_sync(full, l, b);
    if (on && l > lb) f += l - lb;
  }
  const bool cand = on && f <= (long long)c;
  const int lstar = __reduce_max_sync(full, cand ? l : INT_MIN);
  const unsigned who = __ballot_sync(full, cand && l == lstar);
  const int fstar = __shfl_sync(full, (int)f, __ffs(who) - 1);     // f(l*) <= c fits an int
  const unsigned le = __ballot_sync(full, on && l <= lstar);
  const int m = __popc(le);
  const int rest = c - fstar;
  const int lam = lstar + rest / m, rem = rest % m;
  int g = 0;
  if (on && l <= lstar) {
    g = lam - l;
    if (__popc(le & ((1u << lane) - 1u)) < rem) g++;
  }
  if (on) { s.q[j] = g; s.load[r] = l + g; }
  const int changed = __any_sync(full, on && g != qold);
  if (changed) {
    event++;
    if (on && g != qold) s.stamp[r] = event;
  }
  if (lane == 0) s.seen[e] = event;
  __syncwarp();
  return changed;
}

// Phase C: while the lowest max-load rank h reaches (breadth first, ranks expanded through
// replicated experts in ascending expert id, hosts in ascending slot index) a rank with
// load <= max - 2, move one unit along the path.  Run by one lane.
template <typename I>
__device__ __forceinline__ void augment_units(const QuotaSmemT<I> &s, int P, int Ns) {
  for (;;) {
    int mx = INT_MIN, h = 0;
    for (int r = 0; r < P; r++)
      if (s.load[r] > mx) { mx = s.load[r]; h = r; }
    for (int r = 0; r < P; r++) s.visited[r] = 0;
    int head = 0, tail = 0, target = -1;
    s.visited[h] = 1; s.queue[tail++] = h; s.par_rank[h] = -1;
    while (head < tail && target < 0) {
      const int r = s.queue[head++];
      for (int k = 0; k < Ns && target < 0; k++) {
        const int j = s.rslot[r * Ns + k];
        if (j < 0) break;
        const int e = s.se[j];
        if (s.nact[e] < 2 || s.q[j] <= 0) continue;
        const int a0 = s.hptr[e], a1 = a0 + s.nact[e];
        for (int a = a0; a < a1; a++) {
          const int j2 = s.ahs[a], r2 = s.rk[j2];
          if (s.visited[r2]) continue;
          s.visited[r2] = 1; s.par_rank[r2] = r; s.par_from[r2] = j; s.par_to[r2] = j2;
          s.queue[tail++] = r2;
          if (s.load[r2] <= mx - 2) { target = r2; break; }
        }
      }
    }
    if (target < 0) return;
    for (int r2 = target; s.par_rank[r2] >= 0; r2 = s.par_rank[r2]) {
      s.q[s.par_from[r2]] -= 1;
      s.q[s.par_to[r2]] += 1;
    }
    s.load[h] -= 1;
    s.load[target] += 1;
  }
}

// Exclusive scan (in place) of expert e's counts over the chunks [c0, c1) of one instance; returns
// the total = the instance's count of e.
__device__ __forceinline__ int scan_chunk_counts(int32_t *cc, int c0, int c1, int E, int e) {
  int run = 0;
  int c = c0;
  for (; c + 4 <= c1; c += 4) {
    const int v0 = cc[(size_t)c * E + e], v1 = cc[(size_t)(c + 1) * E + e];
    const int v2 = cc[(size_t)(c + 2) * E + e], v3 = cc[(size_t)(c + 3) * E + e];
    cc[(size_t)c * E + e] = run; run += v0;
    cc[(size_t)(c + 1) * E + e] = run; run += v1;
    cc[(size_t)(c + 2) * E + e] = run; run += v2;
    cc[(size_t)(c + 3) * E + e] = run; run += v3;
  }
  for (; c < c1; c++) {
    const int v = cc[(size_t)c * E + e];
    cc[(size_t)c * E + e] = run; run += v;
  }
  return run;
}

template <typename I>
__global__ void __launch_bounds__(kQuotaThreads)
k_quota(const int32_t *__restrict__ hist, const int32_t *__restrict__ quota_in,
        const int32_t *__restrict__ mb_ok, const int32_t *__restrict__ chunk_off,
        const int32_t *__restrict__ pl_host_ptr, const int32_t *__restrict__ pl_host_slot,
        const int32_t *__restrict__ pl_active, const int32_t *__restrict__ pl_rslot,
        const int32_t *__restrict__ pl_fault, const int32_t *__restrict__ slot_expert, int L, int E,
        int P, int Ns, int pl_per_mb, int max_chunks, int32_t *__restrict__ quota,
        int32_t *__restrict__ rank_load, int32_t *__restrict__ slot_off,
        int32_t *__restrict__ inst_cum_end, int32_t *__restrict__ inst_slot_adj,
        int32_t *__restrict__ inst_ok, int32_t *__restrict__ chunk_cnt, int scan_chunks,
        int32_t *dev_status) {
  // scan_chunks: chunk_cnt holds this step's per-chunk counts (the pairs will be assigned)
  extern __shared__ int32_t sm[];
  const int S = P * Ns;
  const int inst = blockIdx.x;
  const int i = inst / L, l = inst - i * L;
  const int pl = pl_per_mb ? inst : l;
  const int tid = threadIdx.x, nt = blockDim.x;
  if (!*mb_ok) return;

  QuotaSmemT<I> s;
  int32_t *p = sm;
  s.c = p; p += E;
  s.seen = p; p += E;
  s.q = p; p += S;
  s.soff = p; p += S + 1;
  s.load = p; p += P;
  s.visited = p; p += P;
  s.par_rank = p; p += P;
  s.par_from = p; p += P;
  s.par_to = p; p += P;
  s.queue = p; p += P;
  s.stamp = p; p += P;
  I *pi = (I *)p;
  s.nact = pi; pi += E;
  s.R = pi; pi += E;
  s.hptr = pi; pi += E + 1;
  s.se = pi; pi += S;
  s.ahs = pi; pi += S;
  s.rk = pi; pi += S;
  s.rslot = pi; pi += S;
  const int32_t *g_hslot = pl_host_slot + (size_t)pl * S;     // used outside the sequential part only
  __shared__ int nR_raw;

  for (int e = tid; e < E; e += nt) s.c[e] = hist[(size_t)inst * E + e];
  for (int e = tid; e <= E; e += nt) s.hptr[e] = pl_host_ptr[(size_t)pl * (E + 1) + e];
  for (int j = tid; j < S; j += nt) {
    int e = slot_expert[(size_t)pl * S + j];
    s.se[j] = (e < -1 || e >= E) ? -1 : e;
    s.rslot[j] = pl_rslot[(size_t)pl * S + j];
    s.rk[j] = j / Ns;
    s.q[j] = 0;
  }
  for (int r = tid; r < P; r += nt) { s.load[r] = 0; s.stamp[r] = 1; }
  for (int e = tid; e < E; e += nt) s.seen[e] = 0;
  if (tid == 0) nR_raw = 0;
  __syncthreads();

  int fault = pl_fault[pl] ? FOREMOE_FAULT_SLOT_EXPERT : 0;
  for (int e = tid; e < E; e += nt) {
    int n = 0;
    for (int a = s.hptr[e]; a < s.hptr[e + 1]; a++) {
      const int j = g_hslot[a];
      if (pl_active[(size_t)pl * S + j]) s.ahs[s.hptr[e] + n++] = j;
    }
    s.nact[e] = n;
    if (s.c[e] < 0) fault |= FOREMOE_FAULT_ID_RANGE;
    if (s.c[e] > 0 && n == 0) fault |= FOREMOE_FAULT_NO_HOST;
  }
  if (quota_in) {
    const int32_t *qi = quota_in + (size_t)inst * S;
    for (int j = tid; j < S; j += nt) {
      const int v = qi[j];
      if (v < 0 || (s.se[j] < 0 && v != 0)) fault |= FOREMOE_FAULT_QUOTA_IN;
      s.q[j] = v;
    }
    for (int e = tid; e < E; e += nt) {
      int64_t sum = 0;
      for (int a = s.hptr[e]; a < s.hptr[e + 1]; a++) sum += qi[g_hslot[a]];
      if (sum != s.c[e]) fault |= FOREMOE_FAULT_QUOTA_IN;
    }
  }
  // every lane of a warp that saw a fault raises it once per warp
  {
    unsigned any = __reduce_or_sync(0xffffffffu, (unsigned)fault);
    if ((tid & 31) == 0 && any) raise_fault(dev_status, (int)any);
  }
  const int any_fault = __syncthreads_or(fault);

  if (any_fault) {
    // outputs of a faulted instance: all-zero plan, pairs get -1
    for (int j = tid; j < S; j += nt) quota[(size_t)inst * S + j] = 0;
    for (int j = tid; j <= S; j += nt) slot_off[(size_t)inst * (S + 1) + j] = 0;
    for (int r = tid; r < P; r += nt) rank_load[(size_t)inst * P + r] = 0;
    if (tid == 0) inst_ok[inst] = 0;
    return;
  }

  if (!quota_in) {
    // Phase A: forced load of singly hosted experts; collect the replicated set
    for (int e = tid; e < E; e += nt) {
      if (s.nact[e] == 1) {
        const int j = s.ahs[s.hptr[e]];
        s.q[j] = s.c[e];
        atomicAdd(&s.load[s.rk[j]], s.c[e]);
      } else if (s.nact[e] >= 2) {
        s.soff[atomicAdd(&nR_raw, 1)] = e;    // soff doubles as the unsorted list (|R| <= S/2)
      }
    }
    __syncthreads();
    const int nR = nR_raw;
    // processing order: descending count, ties ascending expert id (reading 3) -- rank sort
    for (int a = tid; a < nR; a += nt) {
      const int e = s.soff[a], ce = s.c[e];
      int pos = 0;
      for (int b = 0; b < nR; b++) {
        const int e2 = s.soff[b], c2 = s.c[e2];
        pos += (c2 > ce) || (c2 == ce && e2 < e);
      }
      s.R[pos] = e;
    }
    __syncthreads();
    if (tid < 32) {
      // Phase B: Gauss-Seidel water-filling to a fixpoint (warp 0, one lane per host)
      int event = 1;
      for (int pass = 0; pass < kMaxWaterPasses; pass++) {
        int changed = 0;
        for (int a = 0; a < nR; a++) changed |= water_fill_expert_warp(s, s.R[a], tid, event);
        if (!changed) break;
      }
      // Phase C: exactness cleanup
      if (tid == 0) augment_units(s, P, Ns);
    }
  }
  if (tid >= 32 && scan_chunks) {
    // exclusive scan over the instance's chunks, per expert (in place), beside warp 0's quota work
    const int c0 = chunk_off[i], c1 = chunk_off[i + 1];
    int32_t *cc = chunk_cnt + (size_t)l * max_chunks * E;
    for (int e = tid - 32; e < E; e += nt - 32) (void)scan_chunk_counts(cc, c0, c1, E, e);
  }
  __syncthreads();

  // outputs
  if (tid == 0) {
    int run = 0;
    for (int j = 0; j < S; j++) { s.soff[j] = run; run += s.q[j]; }
    s.soff[S] = run;
    inst_ok[inst] = 1;
  }
  __syncthreads();
  for (int j = tid; j < S; j += nt) quota[(size_t)inst * S + j] = s.q[j];
  for (int j = tid; j <= S; j += nt) slot_off[(size_t)inst * (S + 1) + j] = s.soff[j];
  for (int r = tid; r < P; r += nt)
    rank_load[(size_t)inst * P + r] = s.soff[(r + 1) * Ns] - s.soff[r * Ns];
  // pair lookup: a pair of expert e with stable rank n goes to the first host slot j (ascending)
  // with n < cum_end[j]; its row inside the instance is slot_adj[j] + n
  for (int e = tid; e < E; e += nt) {
    int cum = 0;
    for (int a = s.hptr[e]; a < s.hptr[e + 1]; a++) {
      const int j = g_hslot[a];
      inst_slot_adj[(size_t)inst * S + j] = s.soff[j] - cum;
      cum += s.q[j];
      inst_cum_end[(size_t)inst * S + j] = cum;
    }
  }
}

// =============================================================================================
// assign, step 4: stable rank of every pair among its expert's pairs of the instance, then the
// slot (a3) and the destination row (a4).  One CTA per chunk; each warp owns a contiguous segment
// of the chunk, so the order (chunk, warp, iteration, lane) is the (t, k) order.
// grid (max_chunks, L).
//
// Pass 1 (per warp, over its own segment): the rank of every pair among the WARP's pairs of its
// expert, from a warp-private running counter wc[e] and match.any (lanes of one 32-pair group that
// hold the same expert read the same counter, add their position inside the group, and the last of
// them advances it) -- no shared atomics; (expert, rank in warp) stay packed in one register.
// Scan: wc[w][e] -> pairs of e before warp w's segment in the instance (chunk base + earlier warps).
// Pass 2: n = base + rank in warp; etab[e] holds the first host slot of e, where its quota interval
// ends and its row offset: one 16-byte shared load decides every singly hosted expert and the first
// replica.  Pairs beyond the first replica's quota walk htab (one 16-byte entry per further host) in
// a loop whose trip count is uniform over the warp, so the kernel has no divergent branch.
// =============================================================================================
#ifndef FOREMOE_ASSIGN_MINB
#define FOREMOE_ASSIGN_MINB 4
#endif
__global__ void __launch_bounds__(kChunkThreads, FOREMOE_ASSIGN_MINB)
k_assign_pairs(const int32_t *__restrict__ ids, const int32_t *__restrict__ mb_off,
               const int32_t *__restrict__ chunk_off, const int32_t *__restrict__ pl_host_ptr,
               const int32_t *__restrict__ pl_host_slot, const int32_t *__restrict__ inst_cum_end,
               const int32_t *__restrict__ inst_slot_adj, const int32_t *__restrict__ inst_ok,
               const int32_t *__restrict__ chunk_cnt, int L, int T, int K, int E, int S, int n_mb,
               int tpc, int max_chunks, int pl_per_mb, int32_t *__restrict__ pair_slot,
               int32_t *__restrict__ inv, int32_t *dev_status) {
  extern __shared__ __align__(16) int32_t sm_pairs[];
  int4 *etab = (int4 *)sm_pairs;            // [E] {first host slot, its cum_end, its slot_adj, index of the 2nd host or -1}
  int4 *htab = etab + E;                    // [S] per host entry {cum_end, slot, slot_adj, last host of its expert}
  int32_t *wcnt = (int32_t *)(htab + S);    // [kChunkWarps][E]
  ChunkInfo ci;
  const int c = blockIdx.x, l = blockIdx.y;
  if (!locate_chunk(chunk_off, mb_off, n_mb, tpc, c, &ci)) return;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int inst = ci.i * L + l;
  const int pl = pl_per_mb ? inst : l;
  const size_t pbase = ((size_t)l * T + ci.t0) * K;
  const int np = (ci.t1 - ci.t0) * K;
  int32_t *o_slot = pair_slot + pbase, *o_inv = inv + pbase;
  if (!inst_ok[inst]) {
    for (int p = tid; p < np; p += blockDim.x) { o_slot[p] = -1; o_inv[p] = -1; }
    return;
  }
  constexpr int kIter = kChunkPairs / kChunkThreads;   // 32-pair groups per warp
  const int32_t *src = ids + pbase + warp * (kIter * 32) + lane;
  const int rem = np - warp * (kIter * 32) - lane;     // pair `it` of this lane exists iff it * 32 < rem
  int my[kIter];
#pragma unroll
  for (int it = 0; it < kIter; it++) my[it] = it * 32 < rem ? __ldg(src + it * 32) : -1;
  {
    const int32_t *hp = pl_host_ptr + (size_t)pl * (E + 1), *hs = pl_host_slot + (size_t)pl * S;
    const int32_t *ce = inst_cum_end + (size_t)inst * S, *sa = inst_slot_adj + (size_t)inst * S;
    for (int e = tid; e < E; e += blockDim.x) {
      const int a0 = hp[e], a1 = hp[e + 1];
      int4 t = make_int4(-1, 0, 0, -1);
      for (int a = a0; a < a1; a++) {
        const int j = hs[a];
        const int4 h = make_int4(ce[j], j, sa[j], a == a1 - 1);
        htab[a] = h;
        if (a == a0) t = make_int4(j, h.x, h.z, a1 - a0 > 1 ? a0 + 1 : -1);
      }
      etab[e] = t;
    }
  }
  for (int x = tid; x < kChunkWarps * E; x += blockDim.x) wcnt[x] = 0;
  __syncthreads();

  // pass 1: rank inside the warp's segment
  const unsigned full = 0xffffffffu;
  const unsigned lt = (1u << lane) - 1u;
  int32_t *wc = wcnt + warp * E;
  int fault = 0;
#pragma unroll
  for (int it = 0; it < kIter; it++) {
    const int e = my[it];
    const bool ok = (unsigned)e < (unsigned)E;
    // match.any is the kernel's bound (about 37 cycles of the SM's ADU each); ballots over the id bits
    // instead moved the bound to issue slots at the same time per launch (profiles/r02_planner.md)
    const unsigned grp = __match_any_sync(full, ok ? (unsigned)e : (0x80000000u | lane));
    const int pre = wc[ok ? e : 0];
    __syncwarp();
    if (ok && lane == 31 - __clz(grp)) wc[e] = pre + __popc(grp);   // last lane of the group advances the counter
    __syncwarp();
    if (!ok && it * 32 < rem) fault = FOREMOE_FAULT_ID_RANGE;
    my[it] = ok ? (e | ((pre + __popc(grp & lt)) << kRankShift)) : -1;
  }
  __syncthreads();
  // exclusive scan over warps, seeded with the chunk's base (pairs of e in earlier chunks)
  const int32_t *cbase = chunk_cnt + ((size_t)l * max_chunks + c) * E;
  for (int e = tid; e < E; e += blockDim.x) {
    int run = cbase[e];
#pragma unroll
    for (int w = 0; w < kChunkWarps; w++) {
      const int v = wcnt[w * E + e];
      wcnt[w * E + e] = run;
      run += v;
    }
  }
  __syncthreads();

  // pass 2: slot and destination row
  const int row_base = __ldg(mb_off + ci.i) * K;
  o_slot += warp * (kIter * 32) + lane;
  o_inv += warp * (kIter * 32) + lane;
#pragma unroll
  for (int it = 0; it < kIter; it++) {
    const int v = my[it];
    const bool ok = v >= 0;
    const int e = ok ? (v & ((1 << kRankShift) - 1)) : 0;
    const int n = wc[e] + (v >> kRankShift);
    const int4 t = etab[e];
    const bool hit = ok && n < t.y;
    int slot = hit ? t.x : -1;
    int adj = t.z;
    int a = t.w;
    bool pend = ok && !hit && a >= 0;
    while (__any_sync(full, pend)) {            // uniform trip count: the longest host walk of the warp
      const int4 h = htab[pend ? a : 0];
      const bool found = pend && n < h.x;
      if (found) { slot = h.y; adj = h.z; }
      pend = pend && !found && !h.w;
      a++;
    }
    if (ok && slot < 0) fault |= FOREMOE_FAULT_NO_HOST;
    if (it * 32 < rem) {
      o_slot[it * 32] = slot;
      o_inv[it * 32] = slot >= 0 ? row_base + adj + n : -1;
    }
  }
  if (fault) raise_fault(dev_status, fault);
}

// Full serialisation point at the end of foremoe_assign: launched WITHOUT programmatic stream
// serialisation, it starts only when every kernel above has completed and flushed, so a data-path
// kernel that follows (launched with it) can overlap nothing that writes the plan -- the basis of
// FOREMOE_FLAG_PLAN_STABLE's "foremoe_assign excepted".
__global__ void k_plan_fence() {}

}  // namespace foremoe

// =============================================================================================
// C ABI
// =============================================================================================
using namespace foremoe;

namespace foremoe {
int num_sms() {
  static DeviceMemo memo;
  const int dev = current_device();
  int n = memo.get(dev, 0);
  if (n) return n;
  if (dev < 0 || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0)
    return 148;
  memo.put(dev, 0, n);
  return n;
}
}  // namespace foremoe

extern "C" __attribute__((visibility("default"))) int foremoe_version(void) { return 200; }

extern "C" __attribute__((visibility("default"))) int foremoe_workspace_bytes(const foremoe_shape_t *shape, size_t *bytes) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if (!bytes) return FOREMOE_ERR_INVALID_ARG;
  *bytes = make_workspace(d).total;
  return FOREMOE_OK;
}

extern "C" __attribute__((visibility("default"))) int foremoe_load_hist(const foremoe_shape_t *shape, const int32_t *ids,
                                 const int32_t *mb_off, int32_t *hist, int64_t *step_hist,
                                 int32_t *dev_status, void *stream) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if ((!ids && d.T > 0) || !mb_off || !hist) return FOREMOE_ERR_INVALID_ARG;   // T = 0: there are no ids
  cudaStream_t st = (cudaStream_t)stream;
  if (cudaMemsetAsync(hist, 0, sizeof(int32_t) * (size_t)d.n_inst * d.E, st) != cudaSuccess)
    return FOREMOE_ERR_CUDA;
  if (d.T > 0) {
    // tile = 8192 pairs: 32 per thread; the flush is E atomics per tile segment
    const int tile_tokens = (8192 + d.K - 1) / d.K;
    const int tiles_per_layer = (d.T + tile_tokens - 1) / tile_tokens;
    const long long n_tiles = (long long)tiles_per_layer * d.L;
    const int grid = (int)(n_tiles < (long long)num_sms() * 8 ? n_tiles : (long long)num_sms() * 8);
    const size_t smem = sizeof(int32_t) * d.E;
#ifdef FOREMOE_TUNING      // variants 0 / 1 lost the sweep (profiles/r01_hist.md) and exist there only
    if (g_tune.hist_variant == 1)
      k_load_hist<1><<<grid, 256, smem, st>>>(ids, mb_off, d.L, d.T, d.K, d.E, d.n_mb, tile_tokens,
                                              tiles_per_layer, hist, dev_status);
    else if (g_tune.hist_variant == 0)
      k_load_hist<0><<<grid, 256, smem, st>>>(ids, mb_off, d.L, d.T, d.K, d.E, d.n_mb, tile_tokens,
                                              tiles_per_layer, hist, dev_status);
    else
#endif
      k_load_hist<2><<<grid, 256, smem, st>>>(ids, mb_off, d.L, d.T, d.K, d.E, d.n_mb, tile_tokens,
                                              tiles_per_layer, hist, dev_status);
  }
  if (step_hist) {
    const int LE = d.L * d.E;
    k_step_hist<<<(LE + 255) / 256, 256, 0, st>>>(hist, d.n_mb, LE, step_hist);
  }
  return cudaGetLastError() == cudaSuccess ? FOREMOE_OK : FOREMOE_ERR_CUDA;
}

// Shared launcher of foremoe_assign (hist given, hist_out = NULL) and foremoe_plan (hist_out given:
// k_chunk_hist also accumulates the instance histograms and reports the id faults).
static int launch_assign(const Dims &d, const int32_t *ids, const int32_t *mb_off, const int32_t *hist,
                         int32_t *hist_out, int64_t *step_hist, const int32_t *slot_expert,
                         const int32_t *quota_in, int32_t *quota, int32_t *rank_load, int32_t *slot_off,
                         int32_t *pair_slot, int32_t *inv, void *workspace, size_t workspace_bytes,
                         int32_t *dev_status, cudaStream_t st) {
  const bool want_pairs = pair_slot != nullptr;      // both NULL: quotas only (a2), no pass over the ids
  if (!aligned(workspace, 16)) return FOREMOE_ERR_INVALID_ARG;
  const Workspace w = make_workspace(d);
  if (workspace_bytes < w.total) return FOREMOE_ERR_WORKSPACE;
  char *ws = (char *)workspace;
  int32_t *chunk_off = (int32_t *)(ws + w.chunk_off), *mb_ok = (int32_t *)(ws + w.mb_ok);
  int32_t *pl_host_ptr = (int32_t *)(ws + w.pl_host_ptr);
  int32_t *pl_host_slot = (int32_t *)(ws + w.pl_host_slot);
  int32_t *pl_active = (int32_t *)(ws + w.pl_active), *pl_rslot = (int32_t *)(ws + w.pl_rslot);
  int32_t *pl_fault = (int32_t *)(ws + w.pl_fault);
  int32_t *inst_cum_end = (int32_t *)(ws + w.inst_cum_end);
  int32_t *inst_slot_adj = (int32_t *)(ws + w.inst_slot_adj);
  int32_t *inst_ok = (int32_t *)(ws + w.inst_ok), *chunk_cnt = (int32_t *)(ws + w.chunk_cnt);

  // k_quota: int32 arrays c, seen [E], q [S], soff [S+1], 7 x [P]; index arrays nact, R [E], hptr [E+1],
  // se, ahs, rk, rslot [S] as int32 -- or as int16 when that lifts a shared-memory cap on the CTAs per SM
  const size_t q_i32 = (size_t)2 * d.E + (size_t)2 * d.S + 1 + (size_t)7 * d.P;
  const size_t q_idx = (size_t)3 * d.E + 1 + (size_t)4 * d.S;
  const bool quota16 = d.E < 32768 && d.S < 32768 && 4 * (q_i32 + q_idx) * (2048 / kQuotaThreads) > (size_t)kSmemOptIn;
  const size_t smem_quota = 4 * q_i32 + (quota16 ? 2 : 4) * q_idx + 4;
  const size_t smem_pairs = sizeof(int32_t) * ((size_t)4 * d.E + (size_t)4 * d.S + (size_t)kChunkWarps * d.E);
  const size_t smem_pl = sizeof(int32_t) * ((size_t)2 * d.S + d.E + 1);
  if (smem_quota > 200 * 1024 || smem_pairs > 200 * 1024 || smem_pl > 200 * 1024)
    return FOREMOE_ERR_INVALID_ARG;
  if (smem_quota > 48 * 1024 &&
      cudaFuncSetAttribute(quota16 ? k_quota<int16_t> : k_quota<int32_t>,
                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_quota) != cudaSuccess)
    return FOREMOE_ERR_CUDA;
  if (smem_pairs > 48 * 1024 &&
      cudaFuncSetAttribute(k_assign_pairs, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_pairs) != cudaSuccess)
    return FOREMOE_ERR_CUDA;
  if (smem_pl > 48 * 1024 &&
      cudaFuncSetAttribute(k_placement_tables, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_pl) != cudaSuccess)
    return FOREMOE_ERR_CUDA;

  if (hist_out &&
      cudaMemsetAsync(hist_out, 0, sizeof(int32_t) * (size_t)d.n_inst * d.E, st) != cudaSuccess)
    return FOREMOE_ERR_CUDA;        // stays all zero on an MB_OFF fault, like foremoe_load_hist
  k_mb_tables<<<1, 256, 0, st>>>(mb_off, d.n_mb, d.T, d.tpc, chunk_off, mb_ok, dev_status);
  k_placement_tables<<<d.n_pl, 256, smem_pl, st>>>(slot_expert, d.E, d.S, d.Ns, d.P, pl_host_ptr,
                                                   pl_host_slot, pl_active, pl_rslot, pl_fault,
                                                   dev_status);
  const dim3 cgrid(d.max_chunks, d.L);
  const bool chunks = d.T > 0 && want_pairs;
  if (chunks)
    k_chunk_hist<<<cgrid, kChunkThreads, sizeof(int32_t) * d.E, st>>>(
        ids, mb_off, chunk_off, d.L, d.T, d.K, d.E, d.n_mb, d.tpc, d.max_chunks, chunk_cnt, hist_out,
        hist_out ? dev_status : nullptr);
  if (hist_out) hist = hist_out;
  (quota16 ? k_quota<int16_t> : k_quota<int32_t>)<<<d.n_inst, kQuotaThreads, smem_quota, st>>>(
      hist, quota_in, mb_ok, chunk_off, pl_host_ptr, pl_host_slot, pl_active, pl_rslot, pl_fault,
      slot_expert, d.L, d.E, d.P, d.Ns, d.pl_per_mb, d.max_chunks, quota, rank_load, slot_off,
      inst_cum_end, inst_slot_adj, inst_ok, chunk_cnt, chunks ? 1 : 0, dev_status);
  if (hist_out && step_hist) {
    const int LE = d.L * d.E;
    k_step_hist<<<(LE + 255) / 256, 256, 0, st>>>(hist_out, d.n_mb, LE, step_hist);
  }
  if (chunks)
    k_assign_pairs<<<cgrid, kChunkThreads, smem_pairs, st>>>(
        ids, mb_off, chunk_off, pl_host_ptr, pl_host_slot, inst_cum_end, inst_slot_adj, inst_ok,
        chunk_cnt, d.L, d.T, d.K, d.E, d.S, d.n_mb, d.tpc, d.max_chunks, d.pl_per_mb, pair_slot,
        inv, dev_status);
  k_plan_fence<<<1, 32, 0, st>>>();
  return cudaGetLastError() == cudaSuccess ? FOREMOE_OK : FOREMOE_ERR_CUDA;
}

extern "C" __attribute__((visibility("default"))) int foremoe_assign(const foremoe_shape_t *shape, const int32_t *ids,
                              const int32_t *mb_off, const int32_t *hist,
                              const int32_t *slot_expert, const int32_t *quota_in, int32_t *quota,
                              int32_t *rank_load, int32_t *slot_off, int32_t *pair_slot,
                              int32_t *inv, void *workspace, size_t workspace_bytes,
                              int32_t *dev_status, void *stream) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if (!mb_off || !hist || !slot_expert || !quota || !rank_load || !slot_off || !workspace)
    return FOREMOE_ERR_INVALID_ARG;
  if ((pair_slot == nullptr) != (inv == nullptr)) return FOREMOE_ERR_INVALID_ARG;
  // the ids are read only to assign the pairs: quota-only calls (pair_slot = inv = NULL) and steps
  // without tokens may pass ids = NULL, as the header says
  if (!ids && d.T > 0 && pair_slot) return FOREMOE_ERR_INVALID_ARG;
  return launch_assign(d, ids, mb_off, hist, nullptr, nullptr, slot_expert, quota_in, quota, rank_load,
                       slot_off, pair_slot, inv, workspace, workspace_bytes, dev_status, (cudaStream_t)stream);
}

extern "C" __attribute__((visibility("default"))) int foremoe_plan(const foremoe_shape_t *shape, const int32_t *ids,
                            const int32_t *mb_off, const int32_t *slot_expert, const int32_t *quota_in,
                            int32_t *hist, int64_t *step_hist, int32_t *quota, int32_t *rank_load,
                            int32_t *slot_off, int32_t *pair_slot, int32_t *inv, void *workspace,
                            size_t workspace_bytes, int32_t *dev_status, void *stream) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if (!mb_off || !hist || !slot_expert || !quota || !rank_load || !slot_off || !workspace ||
      (d.T > 0 && (!ids || !pair_slot || !inv)))       // T = 0: there are no pairs, the arrays may be NULL
    return FOREMOE_ERR_INVALID_ARG;
  if (d.T == 0) {                                   // no chunks to take the histogram from: all zero
    cudaStream_t st = (cudaStream_t)stream;
    if (cudaMemsetAsync(hist, 0, sizeof(int32_t) * (size_t)d.n_inst * d.E, st) != cudaSuccess ||
        (step_hist && cudaMemsetAsync(step_hist, 0, sizeof(int64_t) * (size_t)d.L * d.E, st) != cudaSuccess))
      return FOREMOE_ERR_CUDA;
    return launch_assign(d, ids, mb_off, hist, nullptr, nullptr, slot_expert, quota_in, quota, rank_load,
                         slot_off, pair_slot, inv, workspace, workspace_bytes, dev_status, st);
  }
  return launch_assign(d, ids, mb_off, nullptr, hist, step_hist, slot_expert, quota_in, quota, rank_load,
                       slot_off, pair_slot, inv, workspace, workspace_bytes, dev_status, (cudaStream_t)stream);
}

// =============================================================================================
// foremoe_plan_noalloc: foremoe_plan for callers that have no device memory to hand over as workspace
// =============================================================================================
// Some users of this library cannot obtain device scratch at the point where they need a plan: a
// component running inside a serving or training engine whose allocator reserved (nearly) all of
// HBM at start-up, so that a cudaMalloc from a guest fails; a plugin whose host forbids allocation
// after initialisation; a step loop that may not pay the device-wide synchronisation a cudaMalloc /
// cudaFree implies.  For them the workspace of the plan kernels lives in the library image itself:
// one fixed array in device global memory, reserved on every GPU that loads the library for as long
// as the process lives.
//
// In host code the name `g_noalloc_scratch` is only a handle the runtime knows the array by -- it is
// NOT the array's device address (handing &g_noalloc_scratch to a kernel would fault, or quietly use
// host memory on systems where the GPU can reach it).  The device address differs per GPU and is
// asked for once per device with cudaGetSymbolAddress, with that device current, and memoised.
static __device__ __align__(256) unsigned char g_noalloc_scratch[FOREMOE_NOALLOC_SCRATCH_BYTES];

static std::atomic<void *> g_noalloc_ptr[foremoe::kMaxDevices];     // zero-initialised: address unknown

// Device address of the scratch array on the calling thread's current device, or NULL on error.
// Two threads that miss together both ask the runtime and store the same address: no lock.
static void *noalloc_scratch_ptr() {
  const int dev = current_device();
  if (dev < 0) return nullptr;
  void *p = g_noalloc_ptr[dev].load(std::memory_order_acquire);
  if (p) return p;
  if (cudaGetSymbolAddress(&p, g_noalloc_scratch) != cudaSuccess || !p) {
    (void)cudaGetLastError();               // do not leave the error sticky for the caller's next call
    return nullptr;
  }
  g_noalloc_ptr[dev].store(p, std::memory_order_release);
  return p;
}

extern "C" __attribute__((visibility("default"))) int foremoe_plan_noalloc(
    const foremoe_shape_t *shape, const int32_t *ids, const int32_t *mb_off, const int32_t *slot_expert,
    const int32_t *quota_in, int32_t *hist, int64_t *step_hist, int32_t *quota, int32_t *rank_load,
    int32_t *slot_off, int32_t *pair_slot, int32_t *inv, int32_t *dev_status, void *stream) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  // the size check comes first and touches no CUDA state: a shape that does not fit is refused
  // before any device is asked for anything
  if (make_workspace(d).total > (size_t)FOREMOE_NOALLOC_SCRATCH_BYTES) return FOREMOE_ERR_WORKSPACE;
  if (!mb_off || !hist || !slot_expert || !quota || !rank_load || !slot_off ||
      (d.T > 0 && (!ids || !pair_slot || !inv)))
    return FOREMOE_ERR_INVALID_ARG;
  void *scratch = noalloc_scratch_ptr();
  if (!scratch) return FOREMOE_ERR_CUDA;
  // No section of the workspace has to start at zero: k_mb_tables, k_placement_tables, k_chunk_hist and
  // k_quota each write every word a later kernel of THIS call reads (the existing entry points are
  // driven with uninitialised workspaces), so what the previous call left behind is never seen.
  return foremoe_plan(shape, ids, mb_off, slot_expert, quota_in, hist, step_hist, quota, rank_load, slot_off,
                      pair_slot, inv, scratch, (size_t)FOREMOE_NOALLOC_SCRATCH_BYTES, dev_status, stream);
}

// Alg. 2 Stage 3: expert replication by a search over (expert, rank) candidates (PAPER.md:337
// sec. 8.2; listing lines 14-19) for every (micro-step, layer) instance.
//   state: every slot holding expert e carries flows x[slot][m] (tokens of e from source machine m);
//   each round every candidate (e, r) -- r has a free redundant slot and does not host e -- is
//   estimated by re-assigning ONLY e's tokens over hosts(e) + r with the locality-aware heuristic
//   (same-machine hosts if the machine has one, else all hosts; least-loaded rank first, ties lowest
//   rank); the smallest Delta of F = a * L_max + b * C_max wins (ties: lowest expert, lowest rank);
//   stop at Delta >= 0 or after P * N_r replicas (reading 40; oracle_replica_search, O16).
// One CTA per instance, one WARP per candidate: lane h holds host h of the expert (hosts are kept
// sorted by rank, the new rank is inserted in place), the token-by-token rule is evaluated in its
// closed form (level by bisection over warp sums, remainder to the lowest eligible lanes), the
// traffic matrix after the move lives in a per-warp scratch.  Candidates that cannot lower F are
// skipped without changing the result: an expert that sits on no most-loaded rank and has no tokens
// on a most-loaded link can only leave L_max and C_max where they are.
// Contract: include/foremoe.h.
#include <limits.h>

#include "foremoe_common.cuh"

namespace foremoe {

namespace {

constexpr int kRsThreads = 256;
constexpr int kRsWarps = kRsThreads / 32;
constexpr unsigned kFull = 0xffffffffu;

__device__ __forceinline__ long long wsum_ll(long long v) {
#pragma unroll
  for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
  return v;
}
__device__ __forceinline__ long long wmax_ll(long long v) {
#pragma unroll
  for (int o = 16; o; o >>= 1) { const long long t = __shfl_xor_sync(kFull, v, o); v = t > v ? t : v; }
  return v;
}
struct RsState {
  int E, P, Ns, Nb, Nr, M, R, maxc;
  long long a, b;
  int32_t *cm;        // [E*M]  c[m][e] at e*M + m
  int32_t *se;        // [S]    current placement
  int32_t *x;         // [S*M]  flows of the slot's expert per source machine
  int32_t *RL;        // [P]
  int32_t *LT;        // [M*M]  LT[i*M + j]: tokens from machine i served on machine j
  int32_t *nhost;     // [E]
  int32_t *nred;      // [P]
  int32_t *hslot;     // [E*maxc] host slots of e, ascending rank
  int32_t *ord;       // [E*M]  source machines of e by descending count, ties ascending m
};

// F after adding a replica of e on rank r_new (all lanes return it).  commit: the estimate becomes
// the state (x, RL, LT, se, host list, counters).  LT2: this warp's [M*M] scratch, flag: its [P] bytes.
__device__ __forceinline__ long long rs_eval(const RsState &s, int e, int r_new, int lane, int32_t *LT2,
                             unsigned char *flag, bool commit) {
  const int M = s.M, Ns = s.Ns, R = s.R, n = s.nhost[e];
  const int32_t *hs = s.hslot + (size_t)e * s.maxc;
  const int rk_old = lane < n ? hs[lane] / Ns : INT_MAX;
  const int pos = __popc(__ballot_sync(kFull, rk_old < r_new));      // lanes before the new host
  const bool isH = lane <= n;
  const int j_new = r_new * Ns + s.Nb + s.nred[r_new];
  int my_slot = -1, my_rank = r_new;
  if (lane < pos) my_slot = hs[lane];
  else if (lane > pos && lane <= n) my_slot = hs[lane - 1];
  if (my_slot >= 0) my_rank = my_slot / Ns;
  int load = 0;                                                      // rank loads stay below 2^31 (T * K < 2^31)
  if (isH) {
    load = s.RL[my_rank];
    if (my_slot >= 0)
      for (int m = 0; m < M; m++) load -= s.x[my_slot * M + m];
  }
  for (int i = lane; i < M * M; i += 32) LT2[i] = s.LT[i];
  __syncwarp();
  if (isH && my_slot >= 0)
    for (int m = 0; m < M; m++) {
      const int v = s.x[my_slot * M + m];
      if (v) atomicSub(LT2 + m * M + my_rank / R, v);
    }
  const int row = my_slot >= 0 ? my_slot : j_new;                    // where this host's flows live
  if (commit && isH)
    for (int m = 0; m < M; m++) s.x[row * M + m] = 0;
  __syncwarp();
  // commodities (e, m) in descending count, ties ascending m (s.ord, fixed per expert); for each the
  // token-by-token rule in closed form: with f(l) = sum over allowed hosts of max(0, l - load), the level
  // sits on top of the highest allowed load l* with f(l*) <= c: lam = l* + (c - f(l*)) / m, m = #{load <= l*},
  // and the (c - f(l*)) % m left-over tokens go one each to the lowest ranks among those m hosts
  const unsigned lanes_lt = (1u << lane) - 1u;
  const unsigned hosts = __ballot_sync(kFull, isH);
  const int my_mach = my_rank / R;
  for (int k = 0; k < M; k++) {
    const int ms = s.ord[e * M + k];
    const int c = s.cm[e * M + ms];
    if (c <= 0) break;
    const unsigned local = __ballot_sync(kFull, isH && my_mach == ms);
    const unsigned allowed = local ? local : hosts;
    const bool al = (allowed >> lane) & 1u;
    long long f = 0;
    for (unsigned mk = allowed; mk; mk &= mk - 1) {
      const int lb = __shfl_sync(kFull, load, __ffs(mk) - 1);
      if (al && load > lb) f += load - lb;
    }
    const bool cand = al && f <= (long long)c;                       // the least-loaded allowed host always is
    const int lstar = __reduce_max_sync(kFull, cand ? load : INT_MIN);
    const int fstar = __shfl_sync(kFull, (int)f, __ffs(__ballot_sync(kFull, cand && load == lstar)) - 1);
    const unsigned le = __ballot_sync(kFull, al && load <= lstar);
    const int m = __popc(le), rest = c - fstar;
    const int lam = lstar + rest / m, rem = rest % m;
    int give = 0;
    if ((le >> lane) & 1u) give = lam - load + (__popc(le & lanes_lt) < rem ? 1 : 0);
    load += give;
    if (give) atomicAdd(LT2 + ms * M + my_mach, give);
    if (commit && give) s.x[row * M + ms] = give;
  }
  __syncwarp();
  // L' = max over all ranks with the hosts' new loads; C' = max off-diagonal of LT2
  if (isH) flag[my_rank] = 1;
  __syncwarp();
  int lmax = isH ? load : INT_MIN;
  for (int r = lane; r < s.P; r += 32)
    if (!flag[r] && s.RL[r] > lmax) lmax = s.RL[r];
  lmax = __reduce_max_sync(kFull, lmax);
  int cmax = 0;
  for (int i = lane; i < M * M; i += 32)
    if (i / M != i % M && LT2[i] > cmax) cmax = LT2[i];
  cmax = __reduce_max_sync(kFull, cmax);
  __syncwarp();
  if (isH) flag[my_rank] = 0;
  if (commit) {
    if (isH) s.RL[my_rank] = load;
    for (int i = lane; i < M * M; i += 32) s.LT[i] = LT2[i];
    __syncwarp();
    if (isH) s.hslot[(size_t)e * s.maxc + lane] = row;               // still ascending rank
    if (lane == 0) {
      s.se[j_new] = e;
      s.nhost[e] = n + 1;
      s.nred[r_new] += 1;
    }
  }
  __syncwarp();
  return s.a * (long long)lmax + s.b * (long long)cmax;
}

}  // namespace

#ifndef FOREMOE_RS_MINB
#define FOREMOE_RS_MINB 4
#endif
__global__ void __launch_bounds__(kRsThreads, FOREMOE_RS_MINB)
k_replica_search(const int32_t *__restrict__ hist_v, const int32_t *__restrict__ placed_se, int L, int E,
                 int P, int Nb, int Nr, int M, int maxc, long long a, long long b,
                 int32_t *__restrict__ out_se, int32_t *__restrict__ replicas_out,
                 long long *__restrict__ F_out, int32_t *dev_status) {
  extern __shared__ int32_t sm[];
  const int Ns = Nb + Nr, S = P * Ns;
  const int inst = blockIdx.x;
  const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, warp = tid >> 5;
  RsState s;
  s.E = E; s.P = P; s.Ns = Ns; s.Nb = Nb; s.Nr = Nr; s.M = M; s.R = P / M; s.maxc = maxc; s.a = a; s.b = b;
  s.cm = sm;
  int32_t *ctot = s.cm + E * M;        // [E]
  s.se = ctot + E;
  s.x = s.se + S;
  s.RL = s.x + S * M;
  s.LT = s.RL + P;
  s.nhost = s.LT + M * M;
  s.nred = s.nhost + E;
  s.hslot = s.nred + P;
  s.ord = s.hslot + E * maxc;
  int32_t *inQ = s.ord + E * M;        // [E]
  const int lt2n = M * M < 2 ? 2 : M * M;
  int32_t *LT2 = inQ + E + warp * lt2n;                                     // [warps][max(M*M, 2)]
  unsigned char *flag = (unsigned char *)(inQ + E + kRsWarps * lt2n) + warp * ((P + 3) / 4 * 4);
  __shared__ int s_fault, s_best_idx;
  __shared__ long long s_best_delta, s_F;
  const int32_t *hv = hist_v + (size_t)inst * E * M;
  const int32_t *pse = placed_se + (size_t)inst * S;
  int32_t *dst = out_se + (size_t)inst * S;

  if (tid == 0) s_fault = 0;
  for (int e = tid; e < E; e += nt) { s.nhost[e] = 0; inQ[e] = 0; }
  for (int r = tid; r < P; r += nt) { s.RL[r] = 0; s.nred[r] = 0; }
  for (int i = tid; i < M * M; i += nt) s.LT[i] = 0;
  for (int i = tid; i < S * M; i += nt) s.x[i] = 0;
  for (int i = tid; i < kRsWarps * ((P + 3) / 4); i += nt) (inQ + E + kRsWarps * lt2n)[i] = 0;
  __syncthreads();
  int fault = 0;
  for (int i = tid; i < E * M; i += nt) {
    const int v = hv[i];
    s.cm[i] = v;
    if (v < 0) fault |= FOREMOE_FAULT_ID_RANGE;
  }
  for (int j = tid; j < S; j += nt) {
    int e = -1;
    if (j % Ns < Nb) {                                   // the input's redundant slots are not read
      e = pse[j];
      if (e < -1 || e >= E) { fault |= FOREMOE_FAULT_SLOT_EXPERT; e = -1; }
      if (e >= 0 && atomicAdd(s.nhost + e, 1) != 0) fault |= FOREMOE_FAULT_SLOT_EXPERT;   // twice in base slots
    }
    s.se[j] = e;
  }
  __syncthreads();
  for (int e = tid; e < E; e += nt) {
    if (s.nhost[e] != 1) fault |= FOREMOE_FAULT_SLOT_EXPERT;
    long long t = 0;
    for (int m = 0; m < M; m++) t += s.cm[e * M + m];
    if (t > INT_MAX) fault |= FOREMOE_FAULT_ID_RANGE;
    ctot[e] = (int)t;
    for (int m = 0; m < M; m++) {                          // position of m in e's processing order
      const int v = s.cm[e * M + m];
      int pos = 0;
      for (int m2 = 0; m2 < M; m2++) {
        const int v2 = s.cm[e * M + m2];
        pos += (v2 > v) || (v2 == v && m2 < m);
      }
      s.ord[e * M + pos] = m;
    }
  }
  if (fault) atomicOr(&s_fault, fault);
  __syncthreads();
  if (s_fault) {
    for (int j = tid; j < S; j += nt) dst[j] = -1;
    if (replicas_out && tid == 0) replicas_out[inst] = 0;
    if (F_out && tid == 0) { F_out[2 * (size_t)inst] = 0; F_out[2 * (size_t)inst + 1] = 0; }
    if (tid == 0) raise_fault(dev_status, s_fault);
    return;
  }
  // initial state: one host per expert, its base slot
  for (int j = tid; j < S; j += nt) {
    const int e = s.se[j];
    if (e < 0) continue;
    const int r = j / Ns;
    s.hslot[(size_t)e * maxc] = j;
    atomicAdd(s.RL + r, ctot[e]);
    for (int m = 0; m < M; m++) {
      const int v = s.cm[e * M + m];
      s.x[j * M + m] = v;
      if (v) atomicAdd(s.LT + m * M + r / s.R, v);
    }
  }
  __syncthreads();

  int placed = 0;
  long long F0 = 0;
  for (int round = 0; round < P * Nr; round++) {
    // ---- F now, and the experts that could lower it -------------------------------------------------
    if (warp == 0) {
      long long lmax = LLONG_MIN, cmax = 0;
      for (int r = lane; r < P; r += 32) lmax = s.RL[r] > lmax ? s.RL[r] : lmax;
      for (int i = lane; i < M * M; i += 32)
        if (i / M != i % M && s.LT[i] > cmax) cmax = s.LT[i];
      lmax = wmax_ll(lmax);
      cmax = wmax_ll(cmax);
      if (lane == 0) {
        s_F = a * lmax + b * cmax;
        s_best_delta = 0;
        s_best_idx = INT_MAX;
        // stash the two maxima for the pruning pass below
        LT2[0] = (int)lmax;
        LT2[1] = (int)cmax;
      }
    }
    __syncthreads();
    const long long F = s_F;
    if (round == 0) F0 = F;
    {
      const int32_t *w0 = inQ + E;                        // warp 0's scratch holds (L_max, C_max)
      const int lmax = w0[0], cmax = w0[1];
      for (int e = tid; e < E; e += nt) {
        int q = 0;
        if (ctot[e] > 0 && s.nhost[e] < maxc)
          for (int h = 0; h < s.nhost[e] && !q; h++) {
            const int j = s.hslot[(size_t)e * maxc + h], r = j / Ns;
            if (s.RL[r] == lmax) q = 1;
            if (b != 0 && cmax > 0)
              for (int m = 0; m < M; m++)
                if (m != r / s.R && s.x[j * M + m] > 0 && s.LT[m * M + r / s.R] == cmax) q = 1;
          }
        inQ[e] = q;
      }
    }
    __syncthreads();
    // ---- candidates: one warp each, (e ascending, r ascending) ------------------------------------
    long long my_delta = 0;
    int my_idx = INT_MAX;
    for (int e = 0; e < E; e++) {
      if (!inQ[e]) continue;
      const int n = s.nhost[e];
      const int hj = lane < n ? s.hslot[(size_t)e * maxc + lane] : -1;
      const int hr = hj >= 0 ? hj / Ns : -1;
      // Lower bounds on F' of every candidate (e, .), so that candidates that cannot beat this warp's best
      // are skipped (a candidate only replaces the best on a STRICTLY smaller Delta, so the result is the
      // same).  Ranks outside hosts(e) + r keep their loads, the loads of hosts(e) + r keep their sum, and a
      // link keeps at least what it carries without e's tokens:
      //   L' >= max(two largest non-host loads as r allows, ceil((sum_hosts RL + RL[r]) / (n + 1)))
      //   C' >= max over links of LT - (e's tokens on the link)
      if (hr >= 0) flag[hr] = 1;
      __syncwarp();
      int t1 = INT_MIN, t1r = -1, t2 = INT_MIN;
      for (int r = lane; r < P; r += 32) {
        if (flag[r]) continue;
        const int v = s.RL[r];
        if (v > t1) { t2 = t1; t1 = v; t1r = r; } else if (v > t2) t2 = v;
      }
      const int g1 = __reduce_max_sync(kFull, t1);
      const int owner = __ffs(__ballot_sync(kFull, t1 == g1)) - 1;
      const int g1r = __shfl_sync(kFull, t1r, owner);
      const int g2 = __reduce_max_sync(kFull, lane == owner ? t2 : t1);
      const long long sumH = wsum_ll(hr >= 0 ? (long long)s.RL[hr] : 0);
      int crest = 0;
      if (b != 0)
        for (int i = lane; i < M * M; i += 32) {
          const int mi = i / M, mj = i % M;
          if (mi == mj) continue;
          int v = s.LT[i];
          for (int h = 0; h < n; h++) {
            const int j = s.hslot[(size_t)e * maxc + h];
            if (j / Ns / s.R == mj) v -= s.x[j * M + mi];
          }
          crest = v > crest ? v : crest;
        }
      crest = __reduce_max_sync(kFull, crest);
      __syncwarp();
      if (hr >= 0) flag[hr] = 0;
      __syncwarp();
      for (int r = warp; r < P; r += kRsWarps) {
        if (s.nred[r] >= Nr) continue;
        if (__any_sync(kFull, hr == r)) continue;
        const long long lrest = r == g1r ? g2 : g1;
        const long long avg = (sumH + s.RL[r] + n) / (n + 1);
        const long long lb = a * (lrest > avg ? lrest : avg) + b * (long long)crest;
        if (lb - F >= my_delta) continue;
        const long long delta = rs_eval(s, e, r, lane, LT2, flag, false) - F;
        if (delta < my_delta) { my_delta = delta; my_idx = e * P + r; }   // strict: first of this warp wins
      }
    }
    if (lane == 0 && my_delta < 0) atomicMin(&s_best_delta, my_delta);
    __syncthreads();
    const long long best_delta = s_best_delta;
    if (best_delta >= 0) break;                           // "if Delta >= 0 then break" (uniform)
    if (lane == 0 && my_delta == best_delta) atomicMin(&s_best_idx, my_idx);
    __syncthreads();
    if (warp == 0) (void)rs_eval(s, s_best_idx / P, s_best_idx % P, lane, LT2, flag, true);
    placed++;
    __syncthreads();
  }
  __syncthreads();
  for (int j = tid; j < S; j += nt) dst[j] = s.se[j];
  if (replicas_out && tid == 0) replicas_out[inst] = placed;
  if (F_out && warp == 0) {
    long long lmax = LLONG_MIN, cmax = 0;
    for (int r = lane; r < P; r += 32) lmax = s.RL[r] > lmax ? s.RL[r] : lmax;
    for (int i = lane; i < M * M; i += 32)
      if (i / M != i % M && s.LT[i] > cmax) cmax = s.LT[i];
    lmax = wmax_ll(lmax);
    cmax = wmax_ll(cmax);
    // N_r = 0: no round ran, F0 was never taken and the state is the initial one: before = after
    if (lane == 0) {
      const long long F1 = a * lmax + b * cmax;
      F_out[2 * (size_t)inst] = P * Nr > 0 ? F0 : F1;
      F_out[2 * (size_t)inst + 1] = F1;
    }
  }
}

}  // namespace foremoe

using namespace foremoe;

extern "C" __attribute__((visibility("default"))) int foremoe_replica_search(
    const foremoe_shape_t *shape, int32_t M, int32_t max_copies, int64_t a, int64_t b, const int32_t *hist_v,
    const int32_t *placed_slot_expert_mb, int32_t *slot_expert_mb, int32_t *replicas, int64_t *F,
    int32_t *dev_status, void *stream) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if (!hist_v || !placed_slot_expert_mb || !slot_expert_mb || M <= 0 || M > 32 || d.P % M != 0 ||
      max_copies < 1 || max_copies > 31 || a < 0 || b < 0 || a > (1 << 20) || b > (1 << 20))
    return FOREMOE_ERR_INVALID_ARG;
  const size_t smem = sizeof(int32_t) * ((size_t)d.E * M + d.E + d.S + (size_t)d.S * M + d.P + (size_t)M * M +
                                         d.E + d.P + (size_t)d.E * max_copies + (size_t)d.E * M + d.E +
                                         (size_t)kRsWarps * (M * M < 2 ? 2 : M * M) +
                                         (size_t)kRsWarps * ((d.P + 3) / 4));
  if (smem > 200 * 1024) return FOREMOE_ERR_INVALID_ARG;
  if (smem > 48 * 1024 &&
      cudaFuncSetAttribute(k_replica_search, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return FOREMOE_ERR_CUDA;
  k_replica_search<<<d.n_inst, kRsThreads, smem, (cudaStream_t)stream>>>(
      hist_v, placed_slot_expert_mb, d.L, d.E, d.P, d.Nb, d.Nr, M, max_copies, (long long)a, (long long)b,
      slot_expert_mb, replicas, (long long *)F, dev_status);
  return cudaGetLastError() == cudaSuccess ? FOREMOE_OK : FOREMOE_ERR_CUDA;
}

// Placements computed from the routing foresight:
//   foremoe_base_placement      Stage 1 at rank level: LPT with N_b base slots per rank
//                               (Alg. 1 lines 13-21; one machine)
//   foremoe_microstep_placement Alg. 3 Stages 2-3 per (micro-step, layer) instance
//                               (PAPER.md:793-819): LPT relocation inside each machine, then
//                               R * N_r rounds of "heaviest local expert -> least-loaded local rank"
// One CTA per problem, one warp per machine; every choice is an integer arg-min / arg-max taken by
// warp reductions, so the result is the oracle's (oracle_base_placement / oracle_microstep_placement)
// bit for bit.  Readings: DESIGN.md sec. 3 (21-25).  Contract: include/foremoe.h.
#include <limits.h>

#include "foremoe_common.cuh"

namespace foremoe {

constexpr int kPlaceThreads = 128;
constexpr unsigned kFull = 0xffffffffu;

__device__ __forceinline__ unsigned long long warp_min_u64(unsigned long long v) {
#pragma unroll
  for (int o = 16; o; o >>= 1) {
    const unsigned long long t = __shfl_xor_sync(kFull, v, o);
    v = t < v ? t : v;
  }
  return v;
}

// exact integer even split of c over n hosts: the idx-th host in ascending slot order
__device__ __forceinline__ int even_share(int c, int n, int idx) { return c / n + (idx < c % n ? 1 : 0); }

struct PlaceSmem {
  int32_t *c, *mach, *order, *copies, *dead, *first, *next, *RL, *nb, *nr, *out, *cntm;
};

// least-loaded rank of machine m among the ranks accepted by `ok(r)`, ties to the lowest rank;
// -1 if none.  All 32 lanes call it.
template <typename Ok>
__device__ __forceinline__ int argmin_rank(const PlaceSmem &s, int r0, int R, int lane, Ok ok) {
  unsigned long long best = ~0ull;
  for (int r = r0 + lane; r < r0 + R; r += 32)
    if (ok(r)) {
      const unsigned long long key = ((unsigned long long)(unsigned)s.RL[r] << 32) | (unsigned)r;
      best = key < best ? key : best;
    }
  best = warp_min_u64(best);
  return best == ~0ull ? -1 : (int)(best & 0xffffffffu);
}

// mode 0: base placement from step totals (no replication); mode 1: Alg. 3 Stages 2-3;
// mode 2: Stage 3 alone on a per-instance placement whose base slots are final (its redundant slots are not read).
__global__ void __launch_bounds__(kPlaceThreads)
k_place(int mode, const int64_t *__restrict__ step_hist, const int32_t *__restrict__ hist,
        const int32_t *__restrict__ base_se, int L, int E, int P, int Nb, int Nr, int M, long long a,
        long long b, int32_t *__restrict__ out_se, int32_t *dev_status) {
  extern __shared__ int32_t sm[];
  const int Ns = Nb + Nr, S = P * Ns, R = P / M;
  const int prob = blockIdx.x;                 // layer (mode 0) or instance i * L + l (mode 1)
  const int l = mode == 0 ? prob : prob % L;
  const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, warp = tid >> 5, nw = nt >> 5;
  PlaceSmem s;
  int32_t *p = sm;
  s.c = p; p += E;
  s.mach = p; p += E;
  s.order = p; p += E;
  s.copies = p; p += E;
  s.dead = p; p += E;
  s.first = p; p += E;
  s.next = p; p += S;
  s.out = p; p += S;
  s.RL = p; p += P;
  s.nb = p; p += P;
  s.nr = p; p += P;
  s.cntm = p; p += M;

  int fault = 0;
  for (int e = tid; e < E; e += nt) {
    long long v = 0;
    if (mode == 0) {               // step totals, per source machine at e*M + m (M = 1: the plain step_hist)
      for (int m = 0; m < M; m++) {
        const long long t = step_hist[((size_t)prob * E + e) * M + m];
        if (t < 0) fault |= FOREMOE_FAULT_ID_RANGE;
        v += t;
      }
    } else {
      v = hist[(size_t)prob * E + e];
    }
    if (v < 0 || v > INT_MAX) { fault |= FOREMOE_FAULT_ID_RANGE; v = 0; }
    s.c[e] = (int)v;
    s.mach[e] = mode == 0 ? 0 : -1;
    s.copies[e] = 0;
    s.dead[e] = 0;
    s.first[e] = INT_MAX;
  }
  for (int j = tid; j < S; j += nt) { s.out[j] = -1; s.next[j] = -1; }
  for (int r = tid; r < P; r += nt) { s.RL[r] = 0; s.nb[r] = 0; s.nr[r] = 0; }
  for (int m = tid; m < M; m += nt) s.cntm[m] = 0;
  __syncthreads();
  if (mode >= 1) {
    // machine of e = machine of its lowest-indexed slot in the base placement
    const int32_t *bse = base_se + (size_t)(mode == 2 ? prob : l) * S;
    for (int j = tid; j < S; j += nt) {
      if (mode == 2 && j % Ns >= Nb) continue;
      const int e = bse[j];
      if (e < -1 || e >= E) fault |= FOREMOE_FAULT_SLOT_EXPERT;
      else if (e >= 0) {
        atomicMin(&s.first[e], j);
        if (mode == 2) atomicAdd(&s.copies[e], 1);       // must end up exactly 1: once in the base slots
      }
    }
    __syncthreads();
    for (int e = tid; e < E; e += nt) {
      if (s.first[e] == INT_MAX || (mode == 2 && s.copies[e] != 1)) { fault |= FOREMOE_FAULT_SLOT_EXPERT; continue; }
      s.mach[e] = (s.first[e] / Ns) / R;
      atomicAdd(&s.cntm[s.mach[e]], 1);
    }
    __syncthreads();
    for (int m = tid; m < M; m += nt)
      if (s.cntm[m] > R * Nb) fault |= FOREMOE_FAULT_SLOT_EXPERT;
  }
  {
    const unsigned any = __reduce_or_sync(kFull, (unsigned)fault);
    if (lane == 0 && any) raise_fault(dev_status, (int)any);
  }
  int32_t *dst = out_se + (size_t)prob * S;
  if (__syncthreads_or(fault)) {
    for (int j = tid; j < S; j += nt) dst[j] = -1;
    return;
  }

  // processing order: descending load, ties ascending id (rank sort)
  for (int e = tid; e < E; e += nt) {
    const int ce = s.c[e];
    int pos = 0;
    for (int e2 = 0; e2 < E; e2++) {
      const int c2 = s.c[e2];
      pos += (c2 > ce) || (c2 == ce && e2 < e);
    }
    s.order[pos] = e;
  }
  __syncthreads();

  if (mode == 0 && M > 1) {
    // Alg. 1 lines 5-12: machine-level greedy, experts in order, one lane per machine (M <= 64):
    // score(m,e) = a*(ML[m] + w_e) + b*(MC[m] + Delta_{m,e}), Delta = w_e - w_{m,e}; machines with a
    // free base slot only (capacity R*Nb); ties to the lowest machine
    __shared__ long long ML[64], MC[64];
    if (warp == 0) {
      for (int m = lane; m < M; m += 32) { ML[m] = 0; MC[m] = 0; }
      __syncwarp();
      for (int x = 0; x < E; x++) {
        const int e = s.order[x];
        const long long we = s.c[e];
        long long best = LLONG_MAX;
        int bm = INT_MAX;
        for (int m = lane; m < M; m += 32) {
          if (s.cntm[m] >= R * Nb) continue;
          const long long wme = step_hist[((size_t)prob * E + e) * M + m];
          const long long sc = a * (ML[m] + we) + b * (MC[m] + we - wme);
          if (sc < best) { best = sc; bm = m; }          // ascending m per lane: strict < keeps the lowest
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) {
          const long long ob = __shfl_xor_sync(kFull, best, o);
          const int om = __shfl_xor_sync(kFull, bm, o);
          if (ob < best || (ob == best && om < bm)) { best = ob; bm = om; }
        }
        if (lane == 0) {
          s.mach[e] = bm;
          s.cntm[bm] += 1;
          ML[bm] += we;
          MC[bm] += we - step_hist[((size_t)prob * E + e) * M + bm];
        }
        __syncwarp();
      }
    }
    __syncthreads();
  }

  for (int m = warp; m < M; m += nw) {
    const int r0 = m * R;
    // Stage 2 / Stage 1: LPT over the machine's ranks with N_b base slots each
    for (int a = 0; a < E; a++) {
      const int e = s.order[a];
      if (s.mach[e] != m) continue;
      // mode 2: the expert keeps the base slot it was given
      const int best = mode == 2 ? s.first[e] / Ns : argmin_rank(s, r0, R, lane, [&](int r) { return s.nb[r] < Nb; });
      if (lane == 0) {
        const int j = mode == 2 ? s.first[e] : best * Ns + s.nb[best];
        s.out[j] = e;
        s.first[e] = j;                  // head of e's host list (ascending slot index)
        s.nb[best] += 1;
        s.RL[best] += s.c[e];
        s.copies[e] = 1;
      }
      __syncwarp();
    }
    if (mode == 0) continue;
    // Stage 3: replication
    for (int k = 0; k < R * Nr; k++) {
      int estar = -1, rstar = -1;
      for (;;) {
        // locally heaviest per copy (exact: cross-multiplied), ties lower id
        int be = INT_MAX, bc = -1, bn = 1;
        for (int e = lane; e < E; e += 32) {
          if (s.mach[e] != m || s.dead[e] || s.c[e] <= 0) continue;
          const long long lhs = (long long)s.c[e] * bn, rhs = (long long)bc * s.copies[e];
          if (be == INT_MAX || lhs > rhs || (lhs == rhs && e < be)) { be = e; bc = s.c[e]; bn = s.copies[e]; }
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) {
          const int oe = __shfl_xor_sync(kFull, be, o), oc = __shfl_xor_sync(kFull, bc, o);
          const int on = __shfl_xor_sync(kFull, bn, o);
          if (oe != INT_MAX) {
            const long long lhs = (long long)oc * bn, rhs = (long long)bc * on;
            if (be == INT_MAX || lhs > rhs || (lhs == rhs && oe < be)) { be = oe; bc = oc; bn = on; }
          }
        }
        if (be == INT_MAX) { estar = -1; break; }
        estar = be;
        rstar = argmin_rank(s, r0, R, lane, [&](int r) {
          if (s.nr[r] >= Nr) return false;
          for (int j = r * Ns; j < (r + 1) * Ns; j++)
            if (s.out[j] == estar) return false;
          return true;
        });
        if (rstar >= 0) break;
        if (lane == 0) s.dead[estar] = 1;        // no eligible rank now => none later either
        __syncwarp();
      }
      if (estar < 0) break;
      if (lane == 0) {
        // RL: even split over n hosts -> even split over n + 1 hosts (hosts in ascending slot index)
        const int ce = s.c[estar], n = s.copies[estar];
        int idx = 0;
        for (int j = s.first[estar]; j >= 0; j = s.next[j]) s.RL[j / Ns] -= even_share(ce, n, idx++);
        const int jn = rstar * Ns + Nb + s.nr[rstar];
        s.out[jn] = estar;
        s.nr[rstar] += 1;
        s.copies[estar] = n + 1;
        if (jn < s.first[estar]) { s.next[jn] = s.first[estar]; s.first[estar] = jn; }
        else {
          int j = s.first[estar];
          while (s.next[j] >= 0 && s.next[j] < jn) j = s.next[j];
          s.next[jn] = s.next[j];
          s.next[j] = jn;
        }
        idx = 0;
        for (int j = s.first[estar]; j >= 0; j = s.next[j]) s.RL[j / Ns] += even_share(ce, n + 1, idx++);
      }
      __syncwarp();
    }
  }
  __syncthreads();
  for (int j = tid; j < S; j += nt) dst[j] = s.out[j];
}

static int launch_place(int mode, const Dims &d, int M, const int64_t *step_hist, const int32_t *hist,
                        const int32_t *base_se, int32_t *out_se, int32_t *dev_status, cudaStream_t st,
                        long long a = 1, long long b = 0) {
  const size_t smem = sizeof(int32_t) * ((size_t)6 * d.E + (size_t)2 * d.S + (size_t)3 * d.P + M);
  if (smem > 200 * 1024) return FOREMOE_ERR_INVALID_ARG;
  if (smem > 48 * 1024 &&
      cudaFuncSetAttribute(k_place, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return FOREMOE_ERR_CUDA;
  const int n_prob = mode == 0 ? d.L : d.n_inst;   // modes 1, 2: one CTA per (micro-step, layer)
  k_place<<<n_prob, kPlaceThreads, smem, st>>>(mode, step_hist, hist, base_se, d.L, d.E, d.P, d.Nb,
                                               d.Nr, M, a, b, out_se, dev_status);
  return cudaGetLastError() == cudaSuccess ? FOREMOE_OK : FOREMOE_ERR_CUDA;
}

}  // namespace foremoe

using namespace foremoe;

extern "C" __attribute__((visibility("default"))) int foremoe_base_placement(
    const foremoe_shape_t *shape, const int64_t *step_hist, int32_t *slot_expert, int32_t *dev_status,
    void *stream) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if (!step_hist || !slot_expert) return FOREMOE_ERR_INVALID_ARG;
  return launch_place(0, d, 1, step_hist, nullptr, nullptr, slot_expert, dev_status, (cudaStream_t)stream);
}

extern "C" __attribute__((visibility("default"))) int foremoe_microstep_placement(
    const foremoe_shape_t *shape, int32_t M, const int32_t *hist, const int32_t *base_slot_expert,
    int32_t *slot_expert_mb, int32_t *dev_status, void *stream) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if (!hist || !base_slot_expert || !slot_expert_mb || M <= 0 || d.P % M != 0)
    return FOREMOE_ERR_INVALID_ARG;
  return launch_place(1, d, M, nullptr, hist, base_slot_expert, slot_expert_mb, dev_status,
                      (cudaStream_t)stream);
}

extern "C" __attribute__((visibility("default"))) int foremoe_replication(
    const foremoe_shape_t *shape, int32_t M, const int32_t *hist, const int32_t *placed_slot_expert_mb,
    int32_t *slot_expert_mb, int32_t *dev_status, void *stream) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if (!hist || !placed_slot_expert_mb || !slot_expert_mb || M <= 0 || d.P % M != 0)
    return FOREMOE_ERR_INVALID_ARG;
  return launch_place(2, d, M, nullptr, hist, placed_slot_expert_mb, slot_expert_mb, dev_status,
                      (cudaStream_t)stream);
}

extern "C" __attribute__((visibility("default"))) int foremoe_base_placement_machines(
    const foremoe_shape_t *shape, int32_t M, int64_t a, int64_t b, const int64_t *step_hist_v,
    int32_t *slot_expert, int32_t *dev_status, void *stream) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if (!step_hist_v || !slot_expert || M <= 0 || M > 64 || d.P % M != 0 || a < 0 || b < 0 ||
      a > (1 << 20) || b > (1 << 20))
    return FOREMOE_ERR_INVALID_ARG;
  return launch_place(0, d, M, step_hist_v, nullptr, nullptr, slot_expert, dev_status, (cudaStream_t)stream,
                      (long long)a, (long long)b);
}

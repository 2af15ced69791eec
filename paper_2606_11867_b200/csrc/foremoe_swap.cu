// Alg. 2 Stage 2: expert relocation by swaps (sec. 8.2; listing lines 4-12,
// PAPER.md:349-372) for every (micro-step, layer) instance -- SURVEY.md sec. 8(f) item 2, second half.
//   each round: h = the bottleneck rank; for every other rank r_l, the `win` heaviest experts on h
//   x the `win` lightest experts on r_l; the swap with the smallest change Delta of
//   F = a * L_max + b * C_max wins (first in enumeration order on ties); stop when Delta >= 0.
// One CTA per instance.  Per round: warp 0 finds h, the three largest rank loads and the three
// largest column maxima of the traffic matrix (so that "max without two ranks / two columns" is a
// lookup); the warps pick the windows by repeated 64-bit arg-max / arg-min shuffles; every thread
// evaluates candidates in O(M); a two-step block reduction (min Delta, then min index among the
// minimisers) reproduces the oracle's "first best wins" bit for bit (oracle_swap_relocation, O12).
// Readings: DESIGN.md 33-35.  Contract: include/foremoe.h.
#include <limits.h>

#include "foremoe_common.cuh"

namespace foremoe {

constexpr int kSwapThreads = 128;
constexpr unsigned kAll = 0xffffffffu;

__device__ __forceinline__ unsigned long long wmax_u64(unsigned long long v) {
#pragma unroll
  for (int o = 16; o; o >>= 1) {
    const unsigned long long t = __shfl_xor_sync(kAll, v, o);
    v = t > v ? t : v;
  }
  return v;
}
__device__ __forceinline__ unsigned long long wmin_u64(unsigned long long v) {
#pragma unroll
  for (int o = 16; o; o >>= 1) {
    const unsigned long long t = __shfl_xor_sync(kAll, v, o);
    v = t < v ? t : v;
  }
  return v;
}

// the three largest values of val[0..n) with their indices (ties: lowest index first), by warp 0;
// results in top_v[3] / top_i[3] (index -1, value INT_MIN when there are fewer than three)
__device__ __forceinline__ void warp_top3(const int32_t *val, int n, int lane, int32_t *top_v, int32_t *top_i) {
  int t0 = -1, t1 = -1;
  for (int k = 0; k < 3; k++) {
    unsigned long long best = 0;
    for (int i = lane; i < n; i += 32) {
      if (i == t0 || i == t1) continue;
      // key: value (biased to unsigned) high, inverted index low -> max = largest value, lowest index
      const unsigned long long key = ((unsigned long long)((unsigned)val[i] ^ 0x80000000u) << 32) |
                                     (unsigned)(0x7fffffff - i);
      best = key > best ? key : best;
    }
    best = wmax_u64(best);
    const int idx = best ? 0x7fffffff - (int)(best & 0xffffffffu) : -1;
    if (lane == 0) {
      top_i[k] = idx;
      top_v[k] = idx >= 0 ? val[idx] : INT_MIN;
    }
    if (k == 0) t0 = idx; else t1 = idx;
  }
}

__device__ __forceinline__ int max_excluding(const int32_t *top_v, const int32_t *top_i, int x, int y) {
#pragma unroll
  for (int k = 0; k < 3; k++)
    if (top_i[k] >= 0 && top_i[k] != x && top_i[k] != y) return top_v[k];
  return INT_MIN;
}

__global__ void __launch_bounds__(kSwapThreads)
k_swap_relocation(const int32_t *__restrict__ hist_v, const int32_t *__restrict__ base_se, int L, int E,
                  int P, int Nb, int Nr, int M, int win, int max_rounds, long long a, long long b,
                  int32_t *__restrict__ out_se, int32_t *__restrict__ rounds_out, int32_t *dev_status) {
  extern __shared__ int32_t sm[];
  const int Ns = Nb + Nr, S = P * Ns, R = P / M, w = win < Nb ? win : Nb;
  const int inst = blockIdx.x, l = inst % L;
  const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, warp = tid >> 5, nw = nt >> 5;
  int32_t *cm = sm;                    // [E*M]  c[m][e] at e*M + m
  int32_t *c = cm + E * M;             // [E]    total load
  int32_t *se = c + E;                 // [S]    current placement
  int32_t *slot_of = se + S;           // [E]
  int32_t *RL = slot_of + E;           // [P]
  int32_t *LT = RL + P;                // [M*M]  LT[i*M + j]: tokens from machine i to machine j
  int32_t *colmax = LT + M * M;        // [M]    max_{i != j} LT[i][j]
  int32_t *heavy = colmax + M;         // [w]
  int32_t *light = heavy + w;          // [P*w]
  int32_t *topR_v = light + P * w, *topR_i = topR_v + 3, *topC_v = topR_i + 3, *topC_i = topC_v + 3;
  __shared__ int s_fault, s_h, s_best_idx;
  __shared__ long long s_best_delta;
  const int32_t *hv = hist_v + (size_t)inst * E * M;
  const int32_t *bse = base_se + (size_t)l * S;
  int32_t *dst = out_se + (size_t)inst * S;

  if (tid == 0) s_fault = 0;
  for (int e = tid; e < E; e += nt) slot_of[e] = -1;
  for (int r = tid; r < P; r += nt) RL[r] = 0;
  for (int i = tid; i < M * M; i += nt) LT[i] = 0;
  __syncthreads();
  int fault = 0;
  for (int i = tid; i < E * M; i += nt) {
    const int v = hv[i];
    cm[i] = v;
    if (v < 0) fault |= FOREMOE_FAULT_ID_RANGE;
  }
  for (int j = tid; j < S; j += nt) {
    const int e = bse[j];
    se[j] = e;
    if (e < -1 || e >= E) { fault |= FOREMOE_FAULT_SLOT_EXPERT; continue; }
    if (e < 0 || j % Ns >= Nb) continue;
    if (atomicCAS(slot_of + e, -1, j) != -1) fault |= FOREMOE_FAULT_SLOT_EXPERT;   // twice in base slots
  }
  __syncthreads();
  for (int e = tid; e < E; e += nt) {
    if (slot_of[e] < 0) fault |= FOREMOE_FAULT_SLOT_EXPERT;
    long long t = 0;
    for (int m = 0; m < M; m++) t += cm[e * M + m];
    if (t > INT_MAX) fault |= FOREMOE_FAULT_ID_RANGE;
    c[e] = (int)t;
  }
  if (fault) atomicOr(&s_fault, fault);
  __syncthreads();
  if (s_fault) {
    for (int j = tid; j < S; j += nt) dst[j] = -1;
    if (rounds_out && tid == 0) rounds_out[inst] = 0;
    if (tid == 0) raise_fault(dev_status, s_fault);
    return;
  }
  // line 3: RL and LT from the placement (one host per expert)
  for (int e = tid; e < E; e += nt) {
    const int r = slot_of[e] / Ns;
    atomicAdd(RL + r, c[e]);
    for (int i = 0; i < M; i++)
      if (cm[e * M + i]) atomicAdd(LT + i * M + r / R, cm[e * M + i]);
  }
  __syncthreads();

  int rounds = 0;
  for (int round = 0; round < max_rounds; round++) {
    // ---- bottleneck rank, top-3 rank loads, column maxima of the traffic matrix -------------------
    for (int j = tid; j < M; j += nt) {
      int mx = INT_MIN;
      for (int i = 0; i < M; i++)
        if (i != j && LT[i * M + j] > mx) mx = LT[i * M + j];
      colmax[j] = mx;                           // INT_MIN when M == 1
    }
    __syncthreads();
    if (warp == 0) {
      warp_top3(RL, P, lane, topR_v, topR_i);
      warp_top3(colmax, M, lane, topC_v, topC_i);
      if (lane == 0) { s_h = topR_i[0]; s_best_delta = 0; s_best_idx = INT_MAX; }
    }
    __syncthreads();
    const int h = s_h;
    // ---- windows: warp 0 the heaviest on h, all warps the lightest on the other ranks ---------
    for (int r = warp; r < P; r += nw) {
      const bool hv_side = r == h;               // heaviest first on h, lightest first elsewhere
      int32_t *wout = hv_side ? heavy : light + r * w;
      unsigned long long prev = 0;
      for (int k = 0; k < w; k++) {
        // keys are distinct (the id sits in the low word) and never 0 / ~0:
        //   heaviest: max of (load, inverted id) below the previous pick
        //   lightest: min of (load, id) above the previous pick
        unsigned long long best = hv_side ? 0ull : ~0ull;
        for (int j = r * Ns + lane; j < r * Ns + Nb; j += 32) {
          const int e = se[j];
          const unsigned long long key = ((unsigned long long)(unsigned)c[e] << 32) |
                                         (unsigned)(hv_side ? 0x7fffffff - e : e);
          if (hv_side) { if ((k == 0 || key < prev) && key > best) best = key; }
          else         { if ((k == 0 || key > prev) && key < best) best = key; }
        }
        best = hv_side ? wmax_u64(best) : wmin_u64(best);
        prev = best;
        const int low = (int)(best & 0xffffffffu);
        if (lane == 0) wout[k] = hv_side ? 0x7fffffff - low : low;
      }
    }
    __syncthreads();
    // ---- candidates: (r_l ascending without h) x heavy x light, enumeration index = idx --------
    const long long Lmax = topR_v[0];
    const long long Cmax = (M > 1 && topC_v[0] > 0) ? topC_v[0] : 0;
    const int n_cand = (P - 1) * w * w;
    long long my_delta = 0;
    int my_idx = INT_MAX;
    for (int idx = tid; idx < n_cand; idx += nt) {
      const int ri = idx / (w * w), x = (idx / w) % w, y = idx % w;
      const int rl = ri < h ? ri : ri + 1;
      const int eh = heavy[x], el = light[rl * w + y];
      const int d = c[el] - c[eh];
      long long lnew = max_excluding(topR_v, topR_i, h, rl);
      const long long nh = (long long)RL[h] + d, nl = (long long)RL[rl] - d;
      lnew = lnew > nh ? lnew : nh;
      lnew = lnew > nl ? lnew : nl;
      long long cnew = Cmax;
      const int mh = h / R, ml = rl / R;
      if (b != 0 && mh != ml) {
        long long mx = max_excluding(topC_v, topC_i, mh, ml);
        for (int i = 0; i < M; i++) {
          const int dd = cm[el * M + i] - cm[eh * M + i];
          if (i != mh) { const long long v = (long long)LT[i * M + mh] + dd; mx = v > mx ? v : mx; }
          if (i != ml) { const long long v = (long long)LT[i * M + ml] - dd; mx = v > mx ? v : mx; }
        }
        cnew = mx > 0 ? mx : 0;
      }
      const long long delta = a * (lnew - Lmax) + b * (cnew - Cmax);
      if (delta < my_delta) { my_delta = delta; my_idx = idx; }     // strict: lowest idx of this thread
    }
    if (my_delta < 0) atomicMin(&s_best_delta, my_delta);
    __syncthreads();
    const long long best_delta = s_best_delta;
    if (best_delta >= 0) break;                  // "if Delta >= 0 then break" (uniform)
    if (my_delta == best_delta) atomicMin(&s_best_idx, my_idx);
    __syncthreads();
    if (tid == 0) {                              // apply the swap, update RL and LT
      const int idx = s_best_idx;
      const int ri = idx / (w * w), x = (idx / w) % w, y = idx % w;
      const int rl = ri < h ? ri : ri + 1;
      const int eh = heavy[x], el = light[rl * w + y];
      const int jh = slot_of[eh], jl = slot_of[el];
      const int d = c[el] - c[eh];
      RL[h] += d; RL[rl] -= d;
      for (int i = 0; i < M; i++) {
        const int dd = cm[el * M + i] - cm[eh * M + i];
        LT[i * M + h / R] += dd;
        LT[i * M + rl / R] -= dd;
      }
      se[jh] = el; se[jl] = eh;
      slot_of[eh] = jl; slot_of[el] = jh;
    }
    rounds++;
    __syncthreads();
  }
  __syncthreads();
  for (int j = tid; j < S; j += nt) dst[j] = se[j];
  if (rounds_out && tid == 0) rounds_out[inst] = rounds;
}

}  // namespace foremoe

using namespace foremoe;

extern "C" __attribute__((visibility("default"))) int foremoe_swap_relocation(
    const foremoe_shape_t *shape, int32_t M, int32_t win, int32_t max_rounds, int64_t a, int64_t b,
    const int32_t *hist_v, const int32_t *base_slot_expert, int32_t *slot_expert_mb, int32_t *rounds,
    int32_t *dev_status, void *stream) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if (!hist_v || !base_slot_expert || !slot_expert_mb || M <= 0 || d.P % M != 0 || win <= 0 ||
      max_rounds < 0 || a < 0 || b < 0 || a > (1 << 20) || b > (1 << 20))
    return FOREMOE_ERR_INVALID_ARG;
  const int w = win < d.Nb ? win : d.Nb;
  const size_t smem = sizeof(int32_t) * ((size_t)d.E * M + 2 * (size_t)d.E + d.S + d.P + (size_t)M * M + M +
                                         w + (size_t)d.P * w + 12);
  if (smem > 200 * 1024) return FOREMOE_ERR_INVALID_ARG;
  if (smem > 48 * 1024 &&
      cudaFuncSetAttribute(k_swap_relocation, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return FOREMOE_ERR_CUDA;
  k_swap_relocation<<<d.n_inst, kSwapThreads, smem, (cudaStream_t)stream>>>(
      hist_v, base_slot_expert, d.L, d.E, d.P, d.Nb, d.Nr, M, win, max_rounds, (long long)a, (long long)b,
      slot_expert_mb, rounds, dev_status);
  return cudaGetLastError() == cudaSuccess ? FOREMOE_OK : FOREMOE_ERR_CUDA;
}

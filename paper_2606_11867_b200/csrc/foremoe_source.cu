// Per-source, multi-machine Stage 4: the locality-aware token
// assignment -- "tokens prefer same-machine replicas to avoid cross-machine traffic, and any
// leftover tokens are routed to minimize per-rank load" -- over w_{s,e} with a source
// per token, and the traffic matrix C_{i,j} of Eq.(5).
//
// The rule is the single-source Stage 4 on COMMODITIES (expert e, source machine m): virtual
// expert v = e*M + m, virtual slot j*M + m (N_s*M per rank) holding v iff slot j is an allowed
// host of (e, m) -- on machine m if that machine holds e, anywhere otherwise (DESIGN.md readings
// 29-31).  So this file only builds the virtual instance; foremoe_load_hist / foremoe_assign /
// foremoe_dispatch / foremoe_combine then run UNCHANGED on the virtual shape
// (E*M, N_b*M, N_r*M): the exact water-filling, the stable ranking and the row movers are reused.
//   foremoe_source_ids       ids_v[l][t][k] = ids[l][t][k]*M + tok_src[t] / (P/M)
//   foremoe_local_placement  slot_expert [n_pl][S] -> slot_expert_v [n_pl][S*M]
//   foremoe_traffic          quota_v [n_mb][L][S*M] -> traffic [n_mb][L][M][M]
// Contract: include/foremoe.h.
#include "foremoe_common.cuh"

namespace foremoe {

// 4 pairs per thread and iteration; tok_src is read through the read-only path (K pairs share it)
__global__ void __launch_bounds__(256)
k_source_ids(const int32_t *__restrict__ ids, const int32_t *__restrict__ tok_src, int L, int T, int K,
             int E, int P, int M, int32_t *__restrict__ ids_v, int32_t *dev_status) {
  const int R = P / M;
  const long long n = (long long)L * T * K;
  const long long TK = (long long)T * K;
  int fault = 0;
  for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < n;
       p += (long long)gridDim.x * blockDim.x) {
    const int t = (int)((p % TK) / K);
    const int e = ids[p];
    const int s = __ldg(tok_src + t);
    int v = -1;
    if (s < 0 || s >= P) fault |= FOREMOE_FAULT_SOURCE;
    else if (e < 0 || e >= E) fault |= FOREMOE_FAULT_ID_RANGE;
    else v = e * M + s / R;
    ids_v[p] = v;
  }
  fault = __reduce_or_sync(0xffffffffu, fault);
  if ((threadIdx.x & 31) == 0) raise_fault(dev_status, fault);
}

// one CTA per placement; smem: holds[E*M] (machine m holds expert e)
__global__ void __launch_bounds__(256)
k_local_placement(const int32_t *__restrict__ se, int E, int S, int Ns, int P, int M,
                  int32_t *__restrict__ se_v, int32_t *dev_status) {
  extern __shared__ int32_t holds[];
  const int R = P / M;
  const int32_t *src = se + (size_t)blockIdx.x * S;
  int32_t *dst = se_v + (size_t)blockIdx.x * S * M;
  for (int i = threadIdx.x; i < E * M; i += blockDim.x) holds[i] = 0;
  __syncthreads();
  int fault = 0;
  for (int j = threadIdx.x; j < S; j += blockDim.x) {
    const int e = src[j];
    if (e < -1 || e >= E) fault |= FOREMOE_FAULT_SLOT_EXPERT;
    else if (e >= 0) holds[e * M + (j / Ns) / R] = 1;
  }
  __syncthreads();
  for (int i = threadIdx.x; i < S * M; i += blockDim.x) {
    const int j = i / M, m = i - j * M;
    const int e = src[j];
    int v = -1;
    if (e >= 0 && e < E && ((j / Ns) / R == m || !holds[e * M + m])) v = e * M + m;
    dst[i] = v;
  }
  raise_fault(dev_status, fault);
}

// one CTA per instance; smem: acc[M*M]
__global__ void __launch_bounds__(256)
k_traffic(const int32_t *__restrict__ quota_v, int S, int Ns, int P, int M,
          int32_t *__restrict__ traffic) {
  extern __shared__ int32_t acc[];
  const int R = P / M;
  const int32_t *q = quota_v + (size_t)blockIdx.x * S * M;
  for (int i = threadIdx.x; i < M * M; i += blockDim.x) acc[i] = 0;
  __syncthreads();
  for (int i = threadIdx.x; i < S * M; i += blockDim.x) {
    const int v = q[i];
    if (v) {
      const int j = i / M, m = i - j * M;
      atomicAdd(acc + m * M + (j / Ns) / R, v);
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < M * M; i += blockDim.x) traffic[(size_t)blockIdx.x * M * M + i] = acc[i];
}

// ---------------------------------------------------------------------------------------------
// Stage 4 under F = a * L_max + b * C_max (Eq.(10)) as a ladder of locality
// thresholds (reading 39).  k_local_placement_theta builds ONE member's virtual placement
// per (micro-step, layer) instance: commodity (e, m) keeps to machine m's copies of e unless
// c[e][m] / n_loc > theta * total / P, i.e. c * den * P > num * n_loc * total (den = 0: never).
// one CTA per instance; smem: nloc[E*M] (ranks of machine m holding e), red[32] (int64 reduction)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_local_placement_theta(const int32_t *__restrict__ se, const int32_t *__restrict__ hist_v, int L, int E,
                        int S, int Ns, int P, int M, int pl_per_mb, long long num, long long den,
                        int32_t *__restrict__ se_v, int32_t *dev_status) {
  extern __shared__ long long red64[];                 // [32] then int32 nloc[E*M]
  int32_t *nloc = (int32_t *)(red64 + 32);
  const int R = P / M, inst = blockIdx.x, l = inst % L;
  const int32_t *src = se + (size_t)(pl_per_mb ? inst : l) * S;
  const int32_t *c = hist_v + (size_t)inst * E * M;
  int32_t *dst = se_v + (size_t)inst * S * M;
  for (int i = threadIdx.x; i < E * M; i += blockDim.x) nloc[i] = 0;
  long long part = 0;
  for (int i = threadIdx.x; i < E * M; i += blockDim.x) part += c[i];
#pragma unroll
  for (int o = 16; o; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
  if ((threadIdx.x & 31) == 0) red64[threadIdx.x >> 5] = part;
  __syncthreads();
  long long total = 0;
  for (int w = 0; w < (int)(blockDim.x >> 5); w++) total += red64[w];
  int fault = 0;
  for (int j = threadIdx.x; j < S; j += blockDim.x) {   // each rank counts an expert once
    const int e = src[j];
    if (e < -1 || e >= E) { fault |= FOREMOE_FAULT_SLOT_EXPERT; continue; }
    if (e < 0) continue;
    bool first = true;
    for (int j2 = (j / Ns) * Ns; j2 < j; j2++) first &= (src[j2] != e);
    if (first) atomicAdd(nloc + e * M + (j / Ns) / R, 1);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < S * M; i += blockDim.x) {
    const int j = i / M, m = i - j * M;
    const int e = src[j];
    int v = -1;
    if (e >= 0 && e < E) {
      const int n = nloc[e * M + m];
      // c < 2^31, den and num <= 2^20, P and n < 2^24, total < 2^31: both products can pass 2^63, so the
      // comparison is made in 128 bits (a wrapped product would silently flip the locality decision)
      const bool spill = n > 0 && den > 0 &&
                         (__int128)c[e * M + m] * den * P > (__int128)num * n * total;
      if ((j / Ns) / R == m || n == 0 || spill) v = e * M + m;
    }
    dst[i] = v;
  }
  raise_fault(dev_status, fault);
}

// The member with the smallest F = a * max_r rank_load + b * max_{i != j} traffic wins (ties: the
// earliest member); its quotas and virtual placement are copied out.  One CTA per instance.
__global__ void __launch_bounds__(256)
k_tradeoff_select(int n_members, size_t n_inst, int P, int M, int SM, long long a, long long b,
                  const int32_t *__restrict__ rank_load_k, const int32_t *__restrict__ traffic_k,
                  const int32_t *__restrict__ quota_k, const int32_t *__restrict__ se_v_k,
                  int32_t *__restrict__ member, long long *__restrict__ F,
                  int32_t *__restrict__ quota_sel, int32_t *__restrict__ se_v_sel) {
  __shared__ int best_k;
  const size_t inst = blockIdx.x;
  if (threadIdx.x == 0) {
    long long best = 0;
    int bk = -1;
    for (int k = 0; k < n_members; k++) {
      const int32_t *rl = rank_load_k + ((size_t)k * n_inst + inst) * P;
      const int32_t *tr = traffic_k + ((size_t)k * n_inst + inst) * M * M;
      long long lmax = 0, cmax = 0;
      for (int r = 0; r < P; r++) lmax = rl[r] > lmax ? rl[r] : lmax;
      for (int i = 0; i < M; i++)
        for (int j = 0; j < M; j++)
          if (i != j && tr[i * M + j] > cmax) cmax = tr[i * M + j];
      const long long f = a * lmax + b * cmax;
      if (F) F[(size_t)k * n_inst + inst] = f;
      if (bk < 0 || f < best) { best = f; bk = k; }
    }
    best_k = bk;
    member[inst] = bk;
  }
  __syncthreads();
  const size_t from = ((size_t)best_k * n_inst + inst) * SM, to = inst * SM;
  for (int i = threadIdx.x; i < SM; i += blockDim.x) {
    quota_sel[to + i] = quota_k[from + i];
    se_v_sel[to + i] = se_v_k[from + i];
  }
}

static int check_machines(const Dims &d, int M) {
  if (M <= 0 || d.P % M != 0) return FOREMOE_ERR_INVALID_ARG;
  if ((int64_t)d.E * M >= ((int64_t)1 << 30) || (int64_t)d.S * M >= ((int64_t)1 << 24))
    return FOREMOE_ERR_INVALID_ARG;
  return FOREMOE_OK;
}

}  // namespace foremoe

using namespace foremoe;

extern "C" __attribute__((visibility("default"))) int foremoe_source_ids(
    const foremoe_shape_t *shape, int32_t M, const int32_t *ids, const int32_t *tok_src,
    int32_t *ids_v, int32_t *dev_status, void *stream) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if ((rc = check_machines(d, M))) return rc;
  if (!ids || !tok_src || !ids_v) return FOREMOE_ERR_INVALID_ARG;
  const long long n = (long long)d.L * d.T * d.K;
  if (n == 0) return FOREMOE_OK;
  long long blocks = (n + 256 * 4 - 1) / (256 * 4);
  const long long cap = (long long)num_sms() * 16;
  if (blocks > cap) blocks = cap;
  k_source_ids<<<(int)blocks, 256, 0, (cudaStream_t)stream>>>(ids, tok_src, d.L, d.T, d.K, d.E, d.P, M,
                                                             ids_v, dev_status);
  return cudaGetLastError() == cudaSuccess ? FOREMOE_OK : FOREMOE_ERR_CUDA;
}

extern "C" __attribute__((visibility("default"))) int foremoe_local_placement(
    const foremoe_shape_t *shape, int32_t M, const int32_t *slot_expert, int32_t *slot_expert_v,
    int32_t *dev_status, void *stream) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if ((rc = check_machines(d, M))) return rc;
  if (!slot_expert || !slot_expert_v) return FOREMOE_ERR_INVALID_ARG;
  const size_t smem = sizeof(int32_t) * (size_t)d.E * M;
  if (smem > 200 * 1024) return FOREMOE_ERR_INVALID_ARG;
  if (smem > 48 * 1024 &&
      cudaFuncSetAttribute(k_local_placement, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return FOREMOE_ERR_CUDA;
  k_local_placement<<<d.n_pl, 256, smem, (cudaStream_t)stream>>>(slot_expert, d.E, d.S, d.Ns, d.P, M,
                                                                 slot_expert_v, dev_status);
  return cudaGetLastError() == cudaSuccess ? FOREMOE_OK : FOREMOE_ERR_CUDA;
}

extern "C" __attribute__((visibility("default"))) int foremoe_traffic(
    const foremoe_shape_t *shape, int32_t M, const int32_t *quota_v, int32_t *traffic, void *stream) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if ((rc = check_machines(d, M))) return rc;
  if (!quota_v || !traffic || M > 128) return FOREMOE_ERR_INVALID_ARG;
  k_traffic<<<d.n_inst, 256, sizeof(int32_t) * (size_t)M * M, (cudaStream_t)stream>>>(
      quota_v, d.S, d.Ns, d.P, M, traffic);
  return cudaGetLastError() == cudaSuccess ? FOREMOE_OK : FOREMOE_ERR_CUDA;
}

extern "C" __attribute__((visibility("default"))) int foremoe_local_placement_theta(
    const foremoe_shape_t *shape, int32_t M, int64_t theta_num, int64_t theta_den, const int32_t *hist_v,
    const int32_t *slot_expert, int32_t *slot_expert_v_mb, int32_t *dev_status, void *stream) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if ((rc = check_machines(d, M))) return rc;
  if (!hist_v || !slot_expert || !slot_expert_v_mb || theta_num < 0 || theta_den < 0 ||
      theta_num > (1 << 20) || theta_den > (1 << 20))
    return FOREMOE_ERR_INVALID_ARG;
  const size_t smem = 32 * sizeof(long long) + sizeof(int32_t) * (size_t)d.E * M;
  if (smem > 200 * 1024) return FOREMOE_ERR_INVALID_ARG;
  if (smem > 48 * 1024 &&
      cudaFuncSetAttribute(k_local_placement_theta, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return FOREMOE_ERR_CUDA;
  k_local_placement_theta<<<d.n_inst, 256, smem, (cudaStream_t)stream>>>(
      slot_expert, hist_v, d.L, d.E, d.S, d.Ns, d.P, M, d.pl_per_mb, theta_num, theta_den,
      slot_expert_v_mb, dev_status);
  return cudaGetLastError() == cudaSuccess ? FOREMOE_OK : FOREMOE_ERR_CUDA;
}

extern "C" __attribute__((visibility("default"))) int foremoe_tradeoff_select(
    const foremoe_shape_t *shape, int32_t M, int32_t n_members, int64_t a, int64_t b,
    const int32_t *rank_load_k, const int32_t *traffic_k, const int32_t *quota_k,
    const int32_t *slot_expert_v_k, int32_t *member, int64_t *F, int32_t *quota_sel,
    int32_t *slot_expert_v_sel, void *stream) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if ((rc = check_machines(d, M))) return rc;
  if (!rank_load_k || !traffic_k || !quota_k || !slot_expert_v_k || !member || !quota_sel ||
      !slot_expert_v_sel || n_members <= 0 || n_members > 64 || a < 0 || b < 0 || a > (1 << 20) ||
      b > (1 << 20) || M > 128)
    return FOREMOE_ERR_INVALID_ARG;
  k_tradeoff_select<<<d.n_inst, 256, 0, (cudaStream_t)stream>>>(
      n_members, (size_t)d.n_inst, d.P, M, d.S * M, a, b, rank_load_k, traffic_k, quota_k,
      slot_expert_v_k, member, (long long *)F, quota_sel, slot_expert_v_sel);
  return cudaGetLastError() == cudaSuccess ? FOREMOE_OK : FOREMOE_ERR_CUDA;
}

// Combine (a6) with a shared-memory ring filled by cp.async (LDGSTS): every thread keeps `D`
// stages of K x 16 bytes in flight in its own shared-memory slots, so the bytes in flight per SM
// are bounded by shared memory (~200 KB) instead of by registers, and the K scattered row reads
// of the next items are always outstanding while the current item is reduced.
//   y[t][h] = fma(w[t][K-1], eo[inv[t*K+K-1]][h], ... fma(w[t][0], eo[inv[t*K]][h], 0))   (fp32)
// One warp per (token, 512-byte slice) item; lane i owns the i-th 16-byte vector of the slice in
// each of the K rows, reads back exactly the bytes it copied (no cross-lane hazard on the data).
#include "foremoe_data.cuh"

namespace foremoe {

// smem: data [D][K][threads] int4, then per warp [D][32] int32 rows and [D][32] float weights
template <bool kBf16, int K_T, int D>
__global__ void __launch_bounds__(512)
k_combine_async(const int32_t *__restrict__ inv_l, const float *__restrict__ w_l,
                const int32_t *__restrict__ mb_off, int mb_begin, int mb_end, int K_rt, int row_vec,
                int n_slices, const int4 *__restrict__ eo, float4 *__restrict__ y) {
  constexpr int kF = kBf16 ? 8 : 4;
  const int K = K_T > 0 ? K_T : K_rt;
  pdl_launch_dependents();
  extern __shared__ __align__(128) unsigned char smem[];
  const int nt = blockDim.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  int4 *data = (int4 *)smem;                                           // [(s*K + k)*nt + tid]
  int32_t *dbuf = (int32_t *)(smem + (size_t)D * K * nt * 16) + warp * D * 32;
  float *wbuf = (float *)(smem + (size_t)D * K * nt * 16 + (size_t)(nt >> 5) * D * 32 * 4) + warp * D * 32;

  const RangeInfo rg = load_range(mb_off, mb_begin, mb_end, K);
  const long long n_items = (long long)(rg.t_end - rg.t_begin) * n_slices;
  const long long W = (long long)gridDim.x * (nt >> 5);
  const long long w0 = (long long)blockIdx.x * (nt >> 5) + warp;
  const int n_my = w0 < n_items ? (int)((n_items - w0 + W - 1) / W) : 0;

  int d_nxt = -1;
  float w_nxt = 0.f;
  auto fetch_meta = [&](int n) {           // inv / w of item n into registers (lanes < K)
    if (n < n_my && lane < K) {
      const long long item = w0 + (long long)n * W;
      const int tl = (int)(item / n_slices);
      const size_t p = (size_t)(rg.t_begin + tl) * K + lane;
      d_nxt = __ldg(inv_l + p);
      w_nxt = w_l ? __ldg(w_l + p) : 1.f;   // w_l == nullptr: unit weights (dispatch backward)
    }
  };
  auto issue = [&](int n) {                // K cp.async of item n into stage n % D
    if (n < n_my) {
      const int s = n % D;
      const long long item = w0 + (long long)n * W;
      const int tl = (int)(item / n_slices);
      const int v = (int)(item - (long long)tl * n_slices) * 32 + lane;
      int d = d_nxt;
      if (lane < K) {
        if (d >= 0) d -= rg.row0;
        dbuf[s * 32 + lane] = d;
        wbuf[s * 32 + lane] = w_nxt;
      }
      fetch_meta(n + 1);
#pragma unroll
      for (int k = 0; k < (K_T > 0 ? K_T : 32); k++) {
        if (K_T == 0 && k >= K) break;
        const int dk = __shfl_sync(0xffffffffu, d, k);
        if (dk >= 0 && v < row_vec)
          cp_async16(smem_u32(data + ((size_t)(s * K + k) * nt + tid)), eo + (size_t)dk * row_vec + v);
      }
    }
    cp_async_commit();
  };

  fetch_meta(0);                           // inv / w / mb_off only: the plan's own arrays (see k_dispatch_rows)
  pdl_wait();                              // expert_out is read and y written after the wait
  for (int n = 0; n < D - 1; n++) issue(n);
  for (int j = 0; j < n_my; j++) {
    issue(j + D - 1);
    cp_async_wait<D - 1>();                // this thread's copies of item j have landed
    __syncwarp();                          // dbuf / wbuf of item j visible to all lanes
    const int s = j % D;
    const long long item = w0 + (long long)j * W;
    const int tl = (int)(item / n_slices);
    const int v = (int)(item - (long long)tl * n_slices) * 32 + lane;
    float acc[kF];
#pragma unroll
    for (int f = 0; f < kF; f++) acc[f] = 0.f;
    if (v < row_vec) {
#pragma unroll
      for (int k = 0; k < (K_T > 0 ? K_T : 32); k++) {
        if (K_T == 0 && k >= K) break;
        const int dk = dbuf[s * 32 + k];
        const float wk = wbuf[s * 32 + k];
        if (dk < 0) continue;
        const int4 r = data[(size_t)(s * K + k) * nt + tid];
        if (kBf16) {
          acc[0] = __fmaf_rn(wk, bf16_lo(r.x), acc[0]);
          acc[1] = __fmaf_rn(wk, bf16_hi(r.x), acc[1]);
          acc[2] = __fmaf_rn(wk, bf16_lo(r.y), acc[2]);
          acc[3] = __fmaf_rn(wk, bf16_hi(r.y), acc[3]);
          acc[4] = __fmaf_rn(wk, bf16_lo(r.z), acc[4]);
          acc[5] = __fmaf_rn(wk, bf16_hi(r.z), acc[5]);
          acc[6] = __fmaf_rn(wk, bf16_lo(r.w), acc[6]);
          acc[7] = __fmaf_rn(wk, bf16_hi(r.w), acc[7]);
        } else {
          acc[0] = __fmaf_rn(wk, __int_as_float(r.x), acc[0]);
          acc[1] = __fmaf_rn(wk, __int_as_float(r.y), acc[1]);
          acc[2] = __fmaf_rn(wk, __int_as_float(r.z), acc[2]);
          acc[3] = __fmaf_rn(wk, __int_as_float(r.w), acc[3]);
        }
      }
      float4 *dst = y + (size_t)tl * row_vec * (kF / 4) + (size_t)v * (kF / 4);
      int4 o;
      o.x = __float_as_int(acc[0]); o.y = __float_as_int(acc[1]);
      o.z = __float_as_int(acc[2]); o.w = __float_as_int(acc[3]);
      st16_stream(dst, o);
      if (kBf16) {
        o.x = __float_as_int(acc[4]); o.y = __float_as_int(acc[5]);
        o.z = __float_as_int(acc[6]); o.w = __float_as_int(acc[7]);
        st16_stream(dst + 1, o);
      }
    }
    __syncwarp();                          // dbuf / wbuf of stage s free before it is refilled
  }
}

template <bool kBf16, int K_T, int D>
static int launch_one(const Dims &d, int threads, const int32_t *inv_l, const float *w_l,
                      const int32_t *mb_off, int mb_begin, int mb_end, const void *eo, float *y,
                      cudaStream_t st) {
  const size_t smem = (size_t)D * d.K * threads * 16 + (size_t)(threads / 32) * D * 32 * 8;
  if (smem > 220 * 1024) return FOREMOE_ERR_INVALID_ARG;
  static int occ = 0, cached_dev = -1;
  static size_t occ_key = 0;
  auto kern = k_combine_async<kBf16, K_T, D>;
  if (cache_stale(&cached_dev)) {
    occ = 0;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024) != cudaSuccess) {
      cached_dev = -1;
      return FOREMOE_ERR_CUDA;
    }
  }
  if (!occ || occ_key != smem * 1024 + threads) { occ = occupancy_ctas(kern, threads, smem); occ_key = smem * 1024 + threads; }
  const int per_sm = g_tune.combine_cta_per_sm > 0 ? g_tune.combine_cta_per_sm : occ;
  const int n_slices = (d.row_vec + 31) / 32;
  const cudaError_t e = launch_pdl(kern, num_sms() * per_sm, threads, smem, st, inv_l, w_l, mb_off,
                                   mb_begin, mb_end, d.K, d.row_vec, n_slices, (const int4 *)eo,
                                   (float4 *)y);
  return e == cudaSuccess ? FOREMOE_OK : FOREMOE_ERR_CUDA;
}

template <bool kBf16, int K_T>
static int launch_depth(int D, const Dims &d, int threads, const int32_t *inv_l, const float *w_l,
                        const int32_t *mb_off, int mb_begin, int mb_end, const void *eo, float *y,
                        cudaStream_t st) {
  switch (D) {
    case 2: return launch_one<kBf16, K_T, 2>(d, threads, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st);
    case 3: return launch_one<kBf16, K_T, 3>(d, threads, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st);
    case 4: return launch_one<kBf16, K_T, 4>(d, threads, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st);
    case 6: return launch_one<kBf16, K_T, 6>(d, threads, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st);
    case 8: return launch_one<kBf16, K_T, 8>(d, threads, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st);
  }
  return FOREMOE_ERR_INVALID_ARG;
}

template <bool kBf16>
static int launch_k(int D, const Dims &d, int threads, const int32_t *inv_l, const float *w_l,
                    const int32_t *mb_off, int mb_begin, int mb_end, const void *eo, float *y,
                    cudaStream_t st) {
  switch (d.K) {
    case 2: return launch_depth<kBf16, 2>(D, d, threads, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st);
    case 8: return launch_depth<kBf16, 8>(D, d, threads, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st);
    case 10: return launch_depth<kBf16, 10>(D, d, threads, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st);
  }
  return launch_depth<kBf16, 0>(D, d, threads, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st);
}

int launch_combine_async(const Dims &d, const int32_t *inv_l, const float *w_l,
                         const int32_t *mb_off, int mb_begin, int mb_end, const void *eo, float *y,
                         cudaStream_t st) {
  // one CTA per SM with up to 512 threads and D >= 2 stages filling <= 190 KB of shared memory
  // (sweep: profiles/r01_sweeps.md): bytes in flight per SM = D * K * threads * 16
  const size_t budget = 190 * 1024;
  int threads = g_tune.combine_threads > 0 ? g_tune.combine_threads : 512;
  if (g_tune.combine_threads <= 0)
    while (threads > 64 && (size_t)2 * d.K * threads * 16 > budget) threads >>= 1;
  int D = g_tune.combine_depth;
  if (D <= 0) {
    const int cand[] = {8, 6, 4, 3, 2};
    D = 2;
    for (int c : cand)
      if ((size_t)c * d.K * threads * 16 <= (threads >= 512 ? 128 * 1024 : budget)) { D = c; break; }
  }
  if (d.act_dtype == FOREMOE_ACT_BF16)
    return launch_k<true>(D, d, threads, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st);
  return launch_k<false>(D, d, threads, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st);
}

}  // namespace foremoe

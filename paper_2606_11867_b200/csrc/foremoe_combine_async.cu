// Combine (a6) with a shared-memory ring filled by cp.async (LDGSTS): every thread keeps `D`
// stages of K x 16 bytes in flight in its own shared-memory slots, so the bytes in flight per SM
// are bounded by shared memory (~200 KB) instead of by registers, and the K scattered row reads
// of the next items are always outstanding while the current item is reduced.
//   y[t][h] = fma(w[t][K-1], eo[inv[t*K+K-1]][h], ... fma(w[t][0], eo[inv[t*K]][h], 0))   (fp32)
// One warp per (token, 512-byte slice) item; lane i owns the i-th 16-byte vector of the slice in
// each of the K rows, reads back exactly the bytes it copied (no cross-lane hazard on the data).
#include "foremoe_data.cuh"

#ifdef FOREMOE_TUNING   // sweep alternative to the bulk-copy ring (combine_impl = 1): not in the product library

namespace foremoe {

// 16-byte cp.async whose source size is 0 when the row is absent: the destination is zero-filled
// and no global access is made, so a skipped pair (inv < 0) or a lane beyond the row needs no branch
__device__ __forceinline__ void cp_async16_zfill(uint32_t dst, const void *src, uint32_t src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" :: "r"(dst), "l"(src), "r"(src_bytes) : "memory");
}

// smem: data [D][K][threads] int4, then per warp [D][32] float weights (0 for a skipped pair).
// Instruction budget matters here: under the board's power cap the SM clock drops to ~1.7 GHz and a
// kernel that keeps the issue slots 60 % busy loses bandwidth with it.  Hence: no divisions in the
// item loop (the (token, slice) cursors advance by a precomputed stride), 32-bit shared-memory byte
// offsets, one 32x32+64-bit multiply-add per global address, zero-fill instead of per-row branches,
// vector loads of the K weights.
template <bool kBf16, int K_T, int D>
__global__ void __launch_bounds__(768)
k_combine_async(const int32_t *__restrict__ inv_l, const float *__restrict__ w_l,
                const int32_t *__restrict__ mb_off, int mb_begin, int mb_end, int K_rt, int row_vec,
                int n_slices, const int4 *__restrict__ eo, float4 *__restrict__ y, int early) {
  constexpr int kF = kBf16 ? 8 : 4;
  constexpr int KU = K_T > 0 ? K_T : 32;
  const int K = K_T > 0 ? K_T : K_rt;
  if (!early) pdl_wait_then_release();     // no global read before the predecessor's writes are visible
  extern __shared__ __align__(128) unsigned char smem[];
  const int nt = blockDim.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = nt >> 5;
  const uint32_t kstride = (uint32_t)nt * 16u, sstride = (uint32_t)K * kstride;       // bytes
  const uint32_t data0 = smem_u32(smem) + (uint32_t)tid * 16u;                        // + s*sstride + k*kstride
  float *wbuf = (float *)(smem + (size_t)D * sstride) + warp * (D * 32);              // [D][32]

  const RangeInfo rg = load_range(mb_off, mb_begin, mb_end, K);
  const long long n_items = (long long)(rg.t_end - rg.t_begin) * n_slices;
  const int W = (int)gridDim.x * nwarp;
  const int w0 = (int)blockIdx.x * nwarp + warp;
  const int n_my = w0 < n_items ? (int)((n_items - w0 + W - 1) / W) : 0;
  const int dW_t = W / n_slices, dW_s = W - dW_t * n_slices;        // cursor stride: one division per kernel
  const uint32_t row_bytes = (uint32_t)row_vec * 16u;

  // three cursors over this warp's items (token, slice): metadata fetch, copy issue, reduce
  int m_tl = w0 / n_slices, m_sl = w0 - m_tl * n_slices;
  int i_tl = m_tl, i_sl = m_sl, c_tl = m_tl, c_sl = m_sl;
  int i_n = 0, i_s = 0, c_s = 0, m_n = 0;
  auto advance = [&](int &tl, int &sl) {
    sl += dW_s; tl += dW_t;
    if (sl >= n_slices) { sl -= n_slices; tl++; }
  };

  int d_nxt = -1;
  float w_nxt = 0.f;
  auto fetch_meta = [&]() {                // inv / w of the next item into registers (lanes < K)
    if (m_n < n_my && lane < K) {
      const size_t p = (size_t)(rg.t_begin + m_tl) * K + lane;
      d_nxt = __ldg(inv_l + p);
      w_nxt = w_l ? __ldg(w_l + p) : 1.f;  // w_l == nullptr: unit weights (dispatch backward)
    }
    m_n++;
    advance(m_tl, m_sl);
  };
  auto issue = [&]() {                     // K cp.async of the next item into stage i_s
    if (i_n < n_my) {
      int d = -1;
      float wv = 0.f;
      if (lane < K && d_nxt >= 0) { d = d_nxt - rg.row0; wv = w_nxt; }
      if (lane < K) wbuf[i_s * 32 + lane] = wv;
      uint32_t voff = (uint32_t)(i_sl * 32 + lane) * 16u;
      const uint32_t sz = voff < row_bytes ? 16u : 0u;      // lanes beyond the row copy nothing
      voff = sz ? voff : 0u;
      fetch_meta();
      const uint32_t dst0 = data0 + (uint32_t)i_s * sstride;
#pragma unroll
      for (int k = 0; k < KU; k++) {
        if (K_T == 0 && k >= K) break;
        const int dk = __shfl_sync(0xffffffffu, d, k);
        const unsigned long long off = (unsigned long long)(unsigned)max(dk, 0) * row_bytes + voff;
        cp_async16_zfill(dst0 + (uint32_t)k * kstride, (const unsigned char *)eo + off, dk >= 0 ? sz : 0u);
      }
      advance(i_tl, i_sl);
      i_s = i_s + 1 == D ? 0 : i_s + 1;
    }
    i_n++;
    cp_async_commit();
  };

  fetch_meta();
  if (early) pdl_wait_then_release();
  for (int n = 0; n < D - 1; n++) issue();
  for (int j = 0; j < n_my; j++) {
    issue();
    cp_async_wait<D - 1>();                // this thread's copies of item j have landed
    __syncwarp();                          // the weights of item j are visible to all lanes
    const uint32_t ds = data0 + (uint32_t)c_s * sstride;
    const float *ws = wbuf + c_s * 32;
    float wk[KU];
    if (K_T > 0 && K_T % 4 == 0) {
#pragma unroll
      for (int q = 0; q < KU / 4; q++) {
        const float4 t = *(const float4 *)(ws + 4 * q);
        wk[4 * q] = t.x; wk[4 * q + 1] = t.y; wk[4 * q + 2] = t.z; wk[4 * q + 3] = t.w;
      }
    } else if (K_T > 0 && K_T % 2 == 0) {
#pragma unroll
      for (int q = 0; q < KU / 2; q++) {
        const float2 t = *(const float2 *)(ws + 2 * q);
        wk[2 * q] = t.x; wk[2 * q + 1] = t.y;
      }
    }
    float acc[kF];
#pragma unroll
    for (int f = 0; f < kF; f++) acc[f] = 0.f;
#pragma unroll
    for (int k = 0; k < KU; k++) {
      if (K_T == 0 && k >= K) break;
      const float w = (K_T > 0 && K_T % 2 == 0) ? wk[k] : ws[k];
      int4 r;
      asm volatile("ld.shared.v4.s32 {%0, %1, %2, %3}, [%4];"
                   : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(ds + (uint32_t)k * kstride));
      if (kBf16) {
        acc[0] = __fmaf_rn(w, bf16_lo(r.x), acc[0]);
        acc[1] = __fmaf_rn(w, bf16_hi(r.x), acc[1]);
        acc[2] = __fmaf_rn(w, bf16_lo(r.y), acc[2]);
        acc[3] = __fmaf_rn(w, bf16_hi(r.y), acc[3]);
        acc[4] = __fmaf_rn(w, bf16_lo(r.z), acc[4]);
        acc[5] = __fmaf_rn(w, bf16_hi(r.z), acc[5]);
        acc[6] = __fmaf_rn(w, bf16_lo(r.w), acc[6]);
        acc[7] = __fmaf_rn(w, bf16_hi(r.w), acc[7]);
      } else {
        acc[0] = __fmaf_rn(w, __int_as_float(r.x), acc[0]);
        acc[1] = __fmaf_rn(w, __int_as_float(r.y), acc[1]);
        acc[2] = __fmaf_rn(w, __int_as_float(r.z), acc[2]);
        acc[3] = __fmaf_rn(w, __int_as_float(r.w), acc[3]);
      }
    }
    const int v = c_sl * 32 + lane;
    if (v < row_vec) {
      float4 *dst = y + ((size_t)c_tl * row_vec + v) * (kF / 4);
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
    advance(c_tl, c_sl);
    c_s = c_s + 1 == D ? 0 : c_s + 1;
    __syncwarp();                          // the stage's weights are free before it is refilled
  }
}

template <bool kBf16, int K_T, int D>
static int launch_one(const Dims &d, int threads, const int32_t *inv_l, const float *w_l,
                      const int32_t *mb_off, int mb_begin, int mb_end, const void *eo, float *y,
                      cudaStream_t st, bool prepare) {
  const size_t smem = (size_t)D * d.K * threads * 16 + (size_t)(threads / 32) * D * 32 * 4;
  if (smem > 220 * 1024) return FOREMOE_ERR_INVALID_ARG;
  auto kern = k_combine_async<kBf16, K_T, D>;
  static DeviceMemo memo;
  const int occ = launch_facts(kern, memo, threads, smem);
  if (!occ) return FOREMOE_ERR_CUDA;
  if (prepare) return FOREMOE_OK;
  const int per_sm = g_tune.combine_cta_per_sm > 0 ? g_tune.combine_cta_per_sm : occ;
  const int n_slices = (d.row_vec + 31) / 32;
  const cudaError_t e = launch_pdl(kern, num_sms() * per_sm, threads, smem, st, inv_l, w_l, mb_off,
                                   mb_begin, mb_end, d.K, d.row_vec, n_slices, (const int4 *)eo,
                                   (float4 *)y, d.plan_stable);
  return e == cudaSuccess ? FOREMOE_OK : FOREMOE_ERR_CUDA;
}

#define FOREMOE_ARGS d, threads, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare

template <bool kBf16, int K_T>
static int launch_depth(int D, const Dims &d, int threads, const int32_t *inv_l, const float *w_l,
                        const int32_t *mb_off, int mb_begin, int mb_end, const void *eo, float *y,
                        cudaStream_t st, bool prepare) {
  switch (D) {
    case 2: return launch_one<kBf16, K_T, 2>(FOREMOE_ARGS);
    case 3: return launch_one<kBf16, K_T, 3>(FOREMOE_ARGS);
    case 4: return launch_one<kBf16, K_T, 4>(FOREMOE_ARGS);
  }
  return FOREMOE_ERR_INVALID_ARG;
}

template <bool kBf16>
static int launch_k(int D, const Dims &d, int threads, const int32_t *inv_l, const float *w_l,
                    const int32_t *mb_off, int mb_begin, int mb_end, const void *eo, float *y,
                    cudaStream_t st, bool prepare) {
  switch (d.K) {
    case 2: return launch_depth<kBf16, 2>(D, FOREMOE_ARGS);
    case 4: return launch_depth<kBf16, 4>(D, FOREMOE_ARGS);
    case 6: return launch_depth<kBf16, 6>(D, FOREMOE_ARGS);
    case 8: return launch_depth<kBf16, 8>(D, FOREMOE_ARGS);
    case 10: return launch_depth<kBf16, 10>(D, FOREMOE_ARGS);
  }
  return launch_depth<kBf16, 0>(D, FOREMOE_ARGS);
}

int launch_combine_async(const Dims &d, const int32_t *inv_l, const float *w_l,
                         const int32_t *mb_off, int mb_begin, int mb_end, const void *eo, float *y,
                         cudaStream_t st, bool prepare) {
  // One CTA per SM, D = 3 stages, about 120 KB of rows in flight: threads = the multiple of 64 with
  // 3 * K * threads * 16 <= 120 KB (K = 8: 320 threads, K = 10: 256).  With the lean instruction
  // stream the kernel is latency-bound, and three shallow stages beat two wide ones on every shape
  // (sweep: profiles/r01_sweeps.md, second addendum).
  int threads = g_tune.combine_threads, D = g_tune.combine_depth;
  if (threads <= 0) {
    threads = (int)(120 * 1024 / ((size_t)(D > 0 ? D : 3) * d.K * 16)) / 64 * 64;
    threads = threads < 64 ? 64 : threads > 512 ? 512 : threads;
  }
  if (D <= 0) {
    D = 3;
    if ((size_t)D * d.K * threads * 16 > 200 * 1024) D = 2;      // K = 32 with 64 threads: 96 KB, fits
  }
  if (d.act_dtype == FOREMOE_ACT_BF16) return launch_k<true>(D, FOREMOE_ARGS);
  return launch_k<false>(D, FOREMOE_ARGS);
}
#undef FOREMOE_ARGS

}  // namespace foremoe

#endif  // FOREMOE_TUNING

// Backward of the data path (the policy-update stage, PAPER.md:241:
// "an additional gradient computation and additional MoE dispatch and MoE combine of gradients",
// run on the SAME plan as the forward, PAPER.md:170 / :188).
//
//   foremoe_combine_bwd   d_eo[inv[t*K+k]][h] = round_act(w[t][k] * dy[t][h])        (token -> slot order)
//                         dw[t][k]           = sum_h dy[t][h] * float(eo[inv[t*K+k]][h])
//   foremoe_dispatch_bwd  dx[t][h] = sum_k float(d_buf[inv[t*K+k]][h]), fp32, k ascending
//                         = the combine kernels with unit weights (foremoe_data.cu / _combine_async.cu)
//
// k_combine_bwd: HBM-bound row mover, no tensor cores (2 flops per 2 bytes moved).  One warp owns a
// TOKEN (all 512-byte slices of its row, so dw[t][:] is reduced inside one warp in a fixed order,
// no atomics); the dy slice and the K scattered eo slices of the next sub-items are pulled with
// cp.async into the thread's own shared-memory slots, D stages deep (same ring as
// k_combine_async), the K scaled rows leave as 16-byte streaming stores.
// Contract: include/foremoe.h; readings: DESIGN.md sec. 3 (26-28).
#include "foremoe_data.cuh"

namespace foremoe {

namespace {

// two fp32 -> packed bf16x2, round to nearest even (lo in bits 0..15)
__device__ __forceinline__ int pack_bf16x2(float lo, float hi) {
  int r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}

// cp.async that copies nothing (zero-fills) when src_bytes == 0: absent rows and lanes beyond the
// row need no branch (same scheme as k_combine_async)
__device__ __forceinline__ void cp_async16_zfill(uint32_t dst, const void *src, uint32_t src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" :: "r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ int4 lds16(uint32_t addr) {
  int4 r;
  asm volatile("ld.shared.v4.s32 {%0, %1, %2, %3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr));
  return r;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

}  // namespace

// smem: data [D][NV][threads] int4 (NV = DY dy vectors + K eo vectors when kDw), then per warp
// [D][32] int32 destination rows and [D][32] float weights.
template <bool kBf16, int K_T, int D, bool kDw>
__global__ void __launch_bounds__(256)
k_combine_bwd(const int32_t *__restrict__ inv_l, const float *__restrict__ w_l,
              const int32_t *__restrict__ mb_off, int mb_begin, int mb_end, int K_rt, int row_vec,
              int n_slices, const int4 *__restrict__ dy, const int4 *__restrict__ eo,
              int4 *__restrict__ d_eo, float *__restrict__ dw_l, int early) {
  constexpr int DY = kBf16 ? 2 : 1;          // 16-byte fp32 vectors of dy per 16-byte row vector
  constexpr int kF = kBf16 ? 8 : 4;
  constexpr int KU = K_T > 0 ? K_T : 32;
  const int K = K_T > 0 ? K_T : K_rt;
  const int NV = DY + (kDw ? K : 0);
  if (!early) pdl_wait_then_release();     // no global read before the predecessor's writes are visible
  extern __shared__ __align__(128) unsigned char smem[];
  const int nt = blockDim.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t vstride = (uint32_t)nt * 16u, sstride = (uint32_t)NV * vstride;   // bytes; slot (s, j) of this thread:
  const uint32_t data0 = smem_u32(smem) + (uint32_t)tid * 16u;                    // data0 + s*sstride + j*vstride
  const uint32_t row_bytes = (uint32_t)row_vec * 16u;
  int32_t *dbuf = (int32_t *)(smem + (size_t)D * NV * nt * 16) + warp * D * 32;
  float *wbuf = (float *)(smem + (size_t)D * NV * nt * 16 + (size_t)(nt >> 5) * D * 32 * 4) + warp * D * 32;

  const RangeInfo rg = load_range(mb_off, mb_begin, mb_end, K);
  const int n_tok = rg.t_end - rg.t_begin;
  const int W = gridDim.x * (nt >> 5);
  const int w0 = blockIdx.x * (nt >> 5) + warp;
  const int n_my = w0 < n_tok ? (n_tok - w0 + W - 1) / W : 0;           // tokens of this warp

  int d_nxt = -1, d_cur = -1;
  float w_nxt = 0.f, w_cur = 0.f;
  auto fetch_meta = [&](int j) {             // inv / w of this warp's j-th token (lanes < K)
    if (j < n_my && lane < K) {
      const size_t p = (size_t)(rg.t_begin + w0 + j * W) * K + lane;
      d_nxt = __ldg(inv_l + p);
      w_nxt = __ldg(w_l + p);
    }
  };
  int i_tok = 0, i_sl = 0, i_n = 0;          // issue cursor: token, slice, sub-item counter
  auto issue = [&]() {
    if (i_tok < n_my) {
      const int s = i_n % D;
      const int tl = w0 + i_tok * W;
      uint32_t voff = (uint32_t)(i_sl * 32 + lane) * 16u;
      const uint32_t sz = voff < row_bytes ? 16u : 0u;          // lanes beyond the row copy nothing
      voff = sz ? voff : 0u;
      if (i_sl == 0) {
        d_cur = d_nxt >= 0 ? d_nxt - rg.row0 : -1;
        w_cur = w_nxt;
        fetch_meta(i_tok + 1);
      }
      if (lane < K) { dbuf[s * 32 + lane] = d_cur; wbuf[s * 32 + lane] = w_cur; }
      const uint32_t dst0 = data0 + (uint32_t)s * sstride;
      const unsigned char *dsrc = (const unsigned char *)dy + ((unsigned long long)(unsigned)tl * row_bytes + voff) * DY;
#pragma unroll
      for (int j = 0; j < DY; j++) cp_async16_zfill(dst0 + (uint32_t)j * vstride, dsrc + 16 * j, sz);
      if (kDw) {
#pragma unroll
        for (int k = 0; k < KU; k++) {
          if (K_T == 0 && k >= K) break;
          const int dk = __shfl_sync(0xffffffffu, d_cur, k);
          const unsigned long long off = (unsigned long long)(unsigned)max(dk, 0) * row_bytes + voff;
          cp_async16_zfill(dst0 + (uint32_t)(DY + k) * vstride, (const unsigned char *)eo + off, dk >= 0 ? sz : 0u);
        }
      }
      i_n++;
      if (++i_sl == n_slices) { i_sl = 0; i_tok++; }
    }
    cp_async_commit();
  };

  float part[KU];
#pragma unroll
  for (int k = 0; k < KU; k++) part[k] = 0.f;

  fetch_meta(0);
  if (early) pdl_wait_then_release();      // only mb_off / inv / w were read (FOREMOE_FLAG_PLAN_STABLE)
  for (int n = 0; n < D - 1; n++) issue();
  int c_n = 0;
  for (int c_tok = 0; c_tok < n_my; c_tok++) {
    const int tl = w0 + c_tok * W;
    for (int c_sl = 0; c_sl < n_slices; c_sl++, c_n++) {
      issue();
      cp_async_wait<D - 1>();              // this thread's copies of sub-item c_n have landed
      __syncwarp();                        // dbuf / wbuf of the stage visible to all lanes
      const int s = c_n % D;
      const int v = c_sl * 32 + lane;
      if (v < row_vec) {
        float g[kF];
        {
          const int4 a = lds16(data0 + (uint32_t)s * sstride);
          g[0] = __int_as_float(a.x); g[1] = __int_as_float(a.y);
          g[2] = __int_as_float(a.z); g[3] = __int_as_float(a.w);
          if (kBf16) {
            const int4 b = lds16(data0 + (uint32_t)s * sstride + vstride);
            g[4] = __int_as_float(b.x); g[5] = __int_as_float(b.y);
            g[6] = __int_as_float(b.z); g[7] = __int_as_float(b.w);
          }
        }
#pragma unroll
        for (int k = 0; k < KU; k++) {
          if (K_T == 0 && k >= K) break;
          const int dk = dbuf[s * 32 + k];
          const float wk = wbuf[s * 32 + k];
          if (dk < 0) continue;
          if (kDw) {
            const int4 r = lds16(data0 + (uint32_t)s * sstride + (uint32_t)(DY + k) * vstride);
            float acc = part[k];
            if (kBf16) {
              acc = __fmaf_rn(g[0], bf16_lo(r.x), acc); acc = __fmaf_rn(g[1], bf16_hi(r.x), acc);
              acc = __fmaf_rn(g[2], bf16_lo(r.y), acc); acc = __fmaf_rn(g[3], bf16_hi(r.y), acc);
              acc = __fmaf_rn(g[4], bf16_lo(r.z), acc); acc = __fmaf_rn(g[5], bf16_hi(r.z), acc);
              acc = __fmaf_rn(g[6], bf16_lo(r.w), acc); acc = __fmaf_rn(g[7], bf16_hi(r.w), acc);
            } else {
              acc = __fmaf_rn(g[0], __int_as_float(r.x), acc); acc = __fmaf_rn(g[1], __int_as_float(r.y), acc);
              acc = __fmaf_rn(g[2], __int_as_float(r.z), acc); acc = __fmaf_rn(g[3], __int_as_float(r.w), acc);
            }
            part[k] = acc;
          }
          int4 o;
          if (kBf16) {
            o.x = pack_bf16x2(__fmul_rn(wk, g[0]), __fmul_rn(wk, g[1]));
            o.y = pack_bf16x2(__fmul_rn(wk, g[2]), __fmul_rn(wk, g[3]));
            o.z = pack_bf16x2(__fmul_rn(wk, g[4]), __fmul_rn(wk, g[5]));
            o.w = pack_bf16x2(__fmul_rn(wk, g[6]), __fmul_rn(wk, g[7]));
          } else {
            o.x = __float_as_int(__fmul_rn(wk, g[0])); o.y = __float_as_int(__fmul_rn(wk, g[1]));
            o.z = __float_as_int(__fmul_rn(wk, g[2])); o.w = __float_as_int(__fmul_rn(wk, g[3]));
          }
          st16_stream((unsigned char *)d_eo + ((unsigned long long)(unsigned)dk * row_bytes + (uint32_t)v * 16u), o);
        }
      }
      __syncwarp();                        // dbuf / wbuf of stage s free before it is refilled
    }
    if (dw_l) {                            // end of the token: dw[t][k] to lane k, one coalesced store
      float mine = 0.f;
#pragma unroll
      for (int k = 0; k < KU; k++) {
        if (K_T == 0 && k >= K) break;
        const float tot = kDw ? warp_sum(part[k]) : 0.f;
        if (lane == k) mine = tot;
        part[k] = 0.f;
      }
      if (lane < K) dw_l[(size_t)(rg.t_begin + tl) * K + lane] = mine;
    }
  }
}

template <bool kBf16, int K_T, int D, bool kDw>
static int launch_one(const Dims &d, int threads, const int32_t *inv_l, const float *w_l, const int32_t *mb_off,
                      int mb_begin, int mb_end, const float *dy, const void *eo, void *d_eo,
                      float *dw_l, cudaStream_t st, bool prepare) {
  const int NV = (kBf16 ? 2 : 1) + (kDw ? d.K : 0);
  const size_t smem = (size_t)D * NV * threads * 16 + (size_t)(threads / 32) * D * 32 * 8;
  if (smem > 220 * 1024) return FOREMOE_ERR_INVALID_ARG;
  auto kern = k_combine_bwd<kBf16, K_T, D, kDw>;
  static DeviceMemo memo;
  const int occ = launch_facts(kern, memo, threads, smem);
  if (!occ) return FOREMOE_ERR_CUDA;
  if (prepare) return FOREMOE_OK;
  // oversubscribed grid: 8-16 CTAs per SM (32 without the eo reads) although only `occ` are resident --
  // fresh CTAs streaming in balance the tail and run 5-9 % faster than a strictly persistent grid
  // (sweep: profiles/r01_backward.md), the same effect as on the dispatch store path
  // size: about one token per warp (mean micro-step of the shape), rounded down to a power of two,
  // at most 16 CTAs per SM with the eo reads (32 without)
  const int cap = kDw ? 16 : 32;
  const long long want = (long long)(d.T / d.n_mb + 1) / ((threads / 32) * (long long)num_sms());
  int dflt = 1;
  while (dflt * 2 <= want && dflt * 2 <= cap) dflt <<= 1;
  const int per_sm = g_tune.bwd_cta_per_sm > 0 ? g_tune.bwd_cta_per_sm : (occ > dflt ? occ : dflt);
  const int n_slices = (d.row_vec + 31) / 32;
  const cudaError_t e = launch_pdl(kern, num_sms() * per_sm, threads, smem, st, inv_l, w_l, mb_off,
                                   mb_begin, mb_end, d.K, d.row_vec, n_slices, (const int4 *)dy,
                                   (const int4 *)eo, (int4 *)d_eo, dw_l, d.plan_stable);
  return e == cudaSuccess ? FOREMOE_OK : FOREMOE_ERR_CUDA;
}

#define FOREMOE_ARGS d, threads, inv_l, w_l, mb_off, mb_begin, mb_end, dy, eo, d_eo, dw_l, st, prepare

template <bool kBf16, int K_T, bool kDw>
static int launch_depth(int D, const Dims &d, int threads, const int32_t *inv_l, const float *w_l,
                        const int32_t *mb_off, int mb_begin, int mb_end, const float *dy,
                        const void *eo, void *d_eo, float *dw_l, cudaStream_t st, bool prepare) {
  switch (D) {
    case 2: return launch_one<kBf16, K_T, 2, kDw>(FOREMOE_ARGS);
    case 3: return launch_one<kBf16, K_T, 3, kDw>(FOREMOE_ARGS);
#ifdef FOREMOE_TUNING      // combine_bwd_rows picks D = 3 (with dw) or 2
    case 4: return launch_one<kBf16, K_T, 4, kDw>(FOREMOE_ARGS);
#endif
  }
  return FOREMOE_ERR_INVALID_ARG;
}

template <bool kBf16, bool kDw>
static int launch_k(int D, const Dims &d, int threads, const int32_t *inv_l, const float *w_l,
                    const int32_t *mb_off, int mb_begin, int mb_end, const float *dy, const void *eo,
                    void *d_eo, float *dw_l, cudaStream_t st, bool prepare) {
  switch (d.K) {
    case 2: return launch_depth<kBf16, 2, kDw>(D, FOREMOE_ARGS);
    case 4: return launch_depth<kBf16, 4, kDw>(D, FOREMOE_ARGS);
    case 6: return launch_depth<kBf16, 6, kDw>(D, FOREMOE_ARGS);
    case 8: return launch_depth<kBf16, 8, kDw>(D, FOREMOE_ARGS);
    case 10: return launch_depth<kBf16, 10, kDw>(D, FOREMOE_ARGS);
  }
  return launch_depth<kBf16, 0, kDw>(D, FOREMOE_ARGS);
}

int combine_bwd_rows(const Dims &d, const int32_t *inv_l, const float *w_l, const int32_t *mb_off,
                     int mb_begin, int mb_end, const float *dy, const void *eo, void *d_eo, float *dw_l,
                     cudaStream_t st, bool want_dw, bool prepare) {
  const int NV = (d.act_dtype == FOREMOE_ACT_BF16 ? 2 : 1) + (want_dw ? d.K : 0);
  // same sizing as k_combine_async: D = 3 stages, about 120 KB in flight per CTA (K = 8: 256 threads,
  // K = 10: 192); without the eo reads only the dy slices are staged and 2 stages of 256 threads do
  int D = g_tune.bwd_depth > 0 ? g_tune.bwd_depth : (want_dw ? 3 : 2);
  int threads = want_dw ? (int)(120 * 1024 / ((size_t)D * NV * 16)) / 32 * 32 : 256;
  threads = threads < 32 ? 32 : threads > 256 ? 256 : threads;
  if (threads > 64) threads = threads / 64 * 64;
  while (D > 2 && (size_t)D * NV * threads * 16 > 200 * 1024) D--;
  const bool bf = d.act_dtype == FOREMOE_ACT_BF16;
  if (bf && want_dw) return launch_k<true, true>(D, FOREMOE_ARGS);
  if (bf) return launch_k<true, false>(D, FOREMOE_ARGS);
  if (want_dw) return launch_k<false, true>(D, FOREMOE_ARGS);
  return launch_k<false, false>(D, FOREMOE_ARGS);
}
#undef FOREMOE_ARGS

}  // namespace foremoe

using namespace foremoe;

extern "C" __attribute__((visibility("default"))) int foremoe_combine_bwd(
    const foremoe_shape_t *shape, int32_t layer, int32_t mb_begin, int32_t mb_end,
    const int32_t *mb_off, const int32_t *inv, const float *w, const float *dy,
    const void *expert_out, void *d_expert_out, float *dw, int32_t *dev_status, void *stream) {
  (void)dev_status;
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if (layer < 0 || layer >= d.L || mb_begin < 0 || mb_end > d.n_mb || mb_begin > mb_end)
    return FOREMOE_ERR_INVALID_ARG;
  if (d.T == 0) return FOREMOE_OK;                     // a step without tokens: the plan arrays may be NULL
  if (!mb_off || !inv || !w || !dy || !d_expert_out || !aligned(dy, 16) ||
      !aligned(d_expert_out, 16) || (expert_out && !aligned(expert_out, 16)))
    return FOREMOE_ERR_INVALID_ARG;
  if (dw && !expert_out) return FOREMOE_ERR_INVALID_ARG;       // dw needs the forward expert outputs
  if (mb_begin == mb_end) return FOREMOE_OK;
  const size_t lo = (size_t)layer * d.T * d.K;
  return combine_bwd_rows(d, inv + lo, w + lo, mb_off, mb_begin, mb_end, dy, expert_out, d_expert_out,
                          dw ? dw + lo : nullptr, (cudaStream_t)stream, dw != nullptr, false);
}

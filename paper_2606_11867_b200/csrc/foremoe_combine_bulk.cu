// Combine (a6) with a bulk-copy (TMA, 1-D) ring: the K scattered row slices of an item are pulled
// into shared memory by K cp.async.bulk copies of 512 B .. 4 KB each (one instruction per slice,
// issued by the lane that holds the row index, completion counted in bytes on an mbarrier), so the
// per-16-byte address arithmetic and LDGSTS issue of the cp.async ring disappear from the
// instruction stream and the kernel no longer follows the SM clock under the board's power cap.
//   y[t][h] = fma(w[t][K-1], eo[inv[t*K+K-1]][h], ... fma(w[t][0], eo[inv[t*K]][h], 0))   (fp32)
// One warp per (token, slice) item, slice = U * 512 bytes of each of the K rows; every warp runs
// its own ring of D stages (nothing is shared between warps, no CTA barrier).  The reduction reads
// the stage with conflict-free 16-byte LDS (lane i owns vector i of every 512-byte piece), runs the
// same fma chain as the other combine kernels (bit-identical result) and stores fp32 with 16-byte
// streaming stores.
#include "foremoe_data.cuh"

namespace foremoe {

namespace {

__device__ __forceinline__ int4 lds16(uint32_t addr) {
  int4 r;
  asm volatile("ld.shared.v4.s32 {%0, %1, %2, %3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr));
  return r;
}
__device__ __forceinline__ void sts16_zero(uint32_t addr) {
  asm volatile("st.shared.v4.s32 [%0], {%1, %1, %1, %1};" :: "r"(addr), "r"(0) : "memory");
}

}  // namespace

// smem: data [warps][D][K][SB] (SB = 512 * U bytes), then per warp [D][32] float weights (0 for a
// skipped pair), then [warps][D] mbarriers.  D <= kMaxDepth stages.
constexpr int kMaxDepth = 4;

template <bool kBf16, int K_T, int U>
__global__ void __launch_bounds__(512)
k_combine_bulk(const int32_t *__restrict__ inv_l, const float *__restrict__ w_l,
               const int32_t *__restrict__ mb_off, int mb_begin, int mb_end, int K_rt, int row_vec,
               int n_slices, int D, const unsigned char *__restrict__ eo, float4 *__restrict__ y, int early) {
  constexpr int kF = kBf16 ? 8 : 4;
  constexpr int KU = K_T > 0 ? K_T : 32;
  constexpr uint32_t SB = 512u * U;
  const int K = K_T > 0 ? K_T : K_rt;
  extern __shared__ __align__(128) unsigned char smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
  const uint32_t stage_bytes = (uint32_t)K * SB;
  const uint32_t data0 = smem_u32(smem) + (uint32_t)(warp * D) * stage_bytes;
  float *wbuf = (float *)(smem + (size_t)(nwarp * D) * stage_bytes) + warp * (D * 32);
  const uint32_t bars0 = smem_u32(smem) + (uint32_t)(nwarp * D) * (stage_bytes + 128u) + (uint32_t)(warp * D) * 8u;

  if (lane == 0)
    for (int s = 0; s < D; s++) mbar_init(bars0 + 8u * s, 1);
  fence_proxy_async();
  __syncwarp();
  if (!early) pdl_wait_then_release();     // no global read before the predecessor's writes are visible

  const RangeInfo rg = load_range(mb_off, mb_begin, mb_end, K);
  const long long n_items = (long long)(rg.t_end - rg.t_begin) * n_slices;
  const int W = (int)gridDim.x * nwarp;
  const int w0 = (int)blockIdx.x * nwarp + warp;
  const int n_my = w0 < n_items ? (int)((n_items - w0 + W - 1) / W) : 0;
  const int dW_t = W / n_slices, dW_s = W - dW_t * n_slices;        // cursor stride: one division per kernel
  const uint32_t row_bytes = (uint32_t)row_vec * 16u;
  const unsigned kmask = K >= 32 ? 0xffffffffu : ((1u << K) - 1u);

  // three cursors over this warp's items (token, slice): metadata fetch, copy issue, reduce
  int m_tl = w0 / n_slices, m_sl = w0 - m_tl * n_slices;
  int i_tl = m_tl, i_sl = m_sl, c_tl = m_tl, c_sl = m_sl;
  int i_n = 0, i_s = 0, c_s = 0, m_n = 0;
  unsigned phase = 0;                      // bit s = parity the next wait on stage s expects
  auto advance = [&](int &tl, int &sl) {
    sl += dW_s; tl += dW_t;
    if (sl >= n_slices) { sl -= n_slices; tl++; }
  };

  int d_nxt = -1;
  float w_nxt = 0.f;
  auto fetch_meta = [&](int &d_out, float &w_out) {   // inv / w of the next item into registers (lanes < K)
    if (m_n < n_my && lane < K) {
      const size_t p = (size_t)(rg.t_begin + m_tl) * K + lane;
      d_out = __ldg(inv_l + p);
      w_out = w_l ? __ldg(w_l + p) : 1.f;  // w_l == nullptr: unit weights (dispatch backward)
    }
    m_n++;
    advance(m_tl, m_sl);
  };
  auto issue = [&](int d_raw, float w_raw) {   // the K bulk copies of the next item into stage i_s
    if (i_n < n_my) {
      int d = -1;
      float wv = 0.f;
      if (lane < K && d_raw >= 0) { d = d_raw - rg.row0; wv = w_raw; }
      if (lane < K) wbuf[i_s * 32 + lane] = wv;
      const uint32_t off = (uint32_t)i_sl * SB;
      const uint32_t bytes = min(SB, row_bytes - off);               // ragged last slice
      const unsigned valid = __ballot_sync(0xffffffffu, d >= 0);
      const uint32_t bar = bars0 + 8u * i_s;
      const uint32_t st0 = data0 + (uint32_t)i_s * stage_bytes;
      if (lane == 0) mbar_expect_tx(bar, bytes * (uint32_t)__popc(valid));
      if (d >= 0)
        bulk_g2s(st0 + (uint32_t)lane * SB, eo + ((unsigned long long)(unsigned)d * row_bytes + off), bytes, bar);
      const unsigned missing = ~valid & kmask;
      if (missing) {                       // rare (faulted pairs): absent rows read as zeros
        for (int k = 0; k < K; k++)
          if ((missing >> k) & 1u)
            for (uint32_t v = lane; v < SB / 16u; v += 32u) sts16_zero(st0 + (uint32_t)k * SB + v * 16u);
        fence_proxy_async();               // before a later bulk copy overwrites these bytes
      }
      advance(i_tl, i_sl);
      i_s = i_s + 1 == D ? 0 : i_s + 1;
    }
    i_n++;
  };

  // prologue: the metadata of the first D items in one round trip, then their copies
  {
    int dq[kMaxDepth];
    float wq[kMaxDepth];
#pragma unroll
    for (int q = 0; q < kMaxDepth; q++) {
      dq[q] = -1; wq[q] = 0.f;
      if (q < D) fetch_meta(dq[q], wq[q]);
    }
    fetch_meta(d_nxt, w_nxt);
    if (early) pdl_wait_then_release();
#pragma unroll
    for (int q = 0; q < kMaxDepth; q++)
      if (q < D) issue(dq[q], wq[q]);
  }
  for (int j = 0; j < n_my; j++) {
    mbar_wait(bars0 + 8u * c_s, (phase >> c_s) & 1u);               // the K slices of item j have landed
    phase ^= 1u << c_s;
    const uint32_t ds = data0 + (uint32_t)c_s * stage_bytes + (uint32_t)lane * 16u;
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
#pragma unroll
    for (int u = 0; u < U; u++) {
      const int v = (c_sl * U + u) * 32 + lane;
      if (v < row_vec) {
        float acc[kF];
#pragma unroll
        for (int f = 0; f < kF; f++) acc[f] = 0.f;
#pragma unroll
        for (int k = 0; k < KU; k++) {
          if (K_T == 0 && k >= K) break;
          const float w = (K_T > 0 && K_T % 2 == 0) ? wk[k] : ws[k];
          const int4 r = lds16(ds + (uint32_t)k * SB + (uint32_t)u * 512u);
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
    }
    advance(c_tl, c_sl);
    c_s = c_s + 1 == D ? 0 : c_s + 1;
    __syncwarp();                          // every lane has read the stage (data and weights): refill it
    issue(d_nxt, w_nxt);
    fetch_meta(d_nxt, w_nxt);
  }
}

template <bool kBf16, int K_T, int U>
static int launch_one(const Dims &d, int warps, int D, const int32_t *inv_l, const float *w_l,
                      const int32_t *mb_off, int mb_begin, int mb_end, const void *eo, float *y,
                      cudaStream_t st, bool prepare) {
  const size_t smem = (size_t)warps * D * ((size_t)d.K * 512 * U + 8 + 128);
  if (smem > 220 * 1024) return FOREMOE_ERR_INVALID_ARG;
  auto kern = k_combine_bulk<kBf16, K_T, U>;
  static DeviceMemo memo;
  const int occ = launch_facts(kern, memo, warps * 32, smem);
  if (!occ) return FOREMOE_ERR_CUDA;
  if (prepare) return FOREMOE_OK;
  const int n_slices = (d.row_vec + 32 * U - 1) / (32 * U);
  int per_sm = g_tune.combine_cta_per_sm;
  if (per_sm <= 0) {      // at least 8 items per warp, between the resident CTAs and 32 per SM (sweep: r02_sweeps.md)
    const long long items = (long long)(d.T / d.n_mb + 1) * n_slices;
    const long long want = items / (8LL * warps * num_sms());
    per_sm = want < occ ? occ : want > 32 ? 32 : (int)want;
  }
  const cudaError_t e = launch_pdl(kern, num_sms() * per_sm, warps * 32, smem, st, inv_l, w_l, mb_off,
                                   mb_begin, mb_end, d.K, d.row_vec, n_slices, D,
                                   (const unsigned char *)eo, (float4 *)y, d.plan_stable);
  return e == cudaSuccess ? FOREMOE_OK : FOREMOE_ERR_CUDA;
}

template <bool kBf16, int K_T>
static int launch_u(int U, const Dims &d, int warps, int D, const int32_t *inv_l, const float *w_l,
                    const int32_t *mb_off, int mb_begin, int mb_end, const void *eo, float *y,
                    cudaStream_t st, bool prepare) {
  switch (U) {
    case 1: return launch_one<kBf16, K_T, 1>(d, warps, D, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
    case 2: return launch_one<kBf16, K_T, 2>(d, warps, D, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
#ifdef FOREMOE_TUNING      // launch_combine_bulk's auto rule picks U = 1 or 2
    case 4: return launch_one<kBf16, K_T, 4>(d, warps, D, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
    case 8: return launch_one<kBf16, K_T, 8>(d, warps, D, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
#endif
  }
  return FOREMOE_ERR_INVALID_ARG;
}

template <bool kBf16>
static int launch_k(int U, const Dims &d, int warps, int D, const int32_t *inv_l, const float *w_l,
                    const int32_t *mb_off, int mb_begin, int mb_end, const void *eo, float *y,
                    cudaStream_t st, bool prepare) {
  switch (d.K) {
    case 2: return launch_u<kBf16, 2>(U, d, warps, D, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
    case 4: return launch_u<kBf16, 4>(U, d, warps, D, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
    case 6: return launch_u<kBf16, 6>(U, d, warps, D, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
    case 8: return launch_u<kBf16, 8>(U, d, warps, D, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
    case 10: return launch_u<kBf16, 10>(U, d, warps, D, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
  }
  return launch_u<kBf16, 0>(U, d, warps, D, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
}

int launch_combine_bulk(const Dims &d, const int32_t *inv_l, const float *w_l,
                        const int32_t *mb_off, int mb_begin, int mb_end, const void *eo, float *y,
                        cudaStream_t st, bool prepare) {
  // Small CTAs on an oversubscribed grid: up to 4 warps x 2 stages of K x 1 KB slices (K = 8: 65 KB of
  // shared memory per CTA, 3 CTAs = 24 stages = 192 KB in flight per SM), up to 32 CTAs per SM in
  // the grid.  SMs drain their share of a bandwidth-bound kernel at rates that differ by ~10 % (ncu:
  // sm__cycles_active min / max of the persistent cp.async ring, profiles/r02_combine.md); with more
  // CTAs than fit, the hardware scheduler hands the faster SMs more of them, and a new CTA's pipeline
  // fill hides behind its neighbours' steady state.  Sweeps on configs 2 / 3 / 5: profiles/r02_sweeps.md.
  const size_t budget = 200 * 1024;
  int U = g_tune.combine_u, D = g_tune.combine_depth, warps = g_tune.combine_threads / 32;
  if (U <= 0) {
    U = 2;
    while (U > 1 && (d.row_bytes < 512 * U || (size_t)2 * 2 * d.K * 512 * U > budget / 2)) U >>= 1;
  }
  if (D <= 0) D = 2;
  if (D > kMaxDepth) D = kMaxDepth;
  const size_t stage = (size_t)d.K * 512 * U + 8 + 128;
  if (warps <= 0) {       // as many warps as let three CTAs share an SM's shared memory (K = 8: 4, K = 10: 3)
    warps = (int)((size_t)kSmemOptIn / 3 / (stage * D));
    warps = warps < 2 ? 2 : warps > 4 ? 4 : warps;
  }
  if (warps > 16) warps = 16;
  while (warps > 1 && stage * D * warps > budget) warps--;
  while (D > 2 && stage * D * warps > budget) D--;
  if (stage * D * warps > 220 * 1024) return FOREMOE_ERR_INVALID_ARG;
  if (d.act_dtype == FOREMOE_ACT_BF16)
    return launch_k<true>(U, d, warps, D, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
  return launch_k<false>(U, d, warps, D, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
}

}  // namespace foremoe

// Data-path kernels of the ForeMoE hot path (sm_100a): dispatch = permutation + row gather (a4/a5)
// and the weighted top-K combine (a6).  HBM-bound row movers: no tensor cores (nothing here is a
// dense contraction), 16-byte vectors, whole rows contiguous, persistent grids sized from the SM
// count.  Contract: include/foremoe.h.
#include "foremoe_data.cuh"

namespace foremoe {

// =============================================================================================
// a4 + a5: dispatch.  Token-major: the row of token t is read ONCE and stored to its K
// destination rows inv[t*K + k] (reading x once matters when x does not fit L2, e.g. H = 7168).
// One warp per (token, slice) item, slice = 32 * U 16-byte vectors; U loads in flight per lane,
// then K * U stores.  perm[inv[p] - row0] = p is scattered by the lanes that hold inv.
// =============================================================================================
template <int U>
__global__ void __launch_bounds__(256)
k_dispatch_rows(const int32_t *__restrict__ inv_l, const int32_t *__restrict__ mb_off, int mb_begin,
                int mb_end, int K, int row_vec, int n_slices, const int4 *__restrict__ x,
                int32_t *__restrict__ perm, int4 *__restrict__ buf, int early) {
  // Nothing in global memory is read before the grid-dependency wait: CUDA guarantees the
  // predecessor's writes (inv from foremoe_assign, x from the caller's kernel) only after it.
  if (!early) pdl_wait_then_release();
  const RangeInfo rg = load_range(mb_off, mb_begin, mb_end, K);
  const int lane = threadIdx.x & 31;
  const long long n_items = (long long)(rg.t_end - rg.t_begin) * n_slices;
  const long long warps = (long long)gridDim.x * (blockDim.x >> 5);
  const long long item0 = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  int d_first = -1;
  if (early) {
    if (item0 < n_items && lane < K) d_first = __ldg(inv_l + (rg.t_begin + (int)(item0 / n_slices)) * K + lane);
    pdl_wait_then_release();
  }
  for (long long item = item0; item < n_items; item += warps) {
    const int tl = (int)(item / n_slices);
    const int sl = (int)(item - (long long)tl * n_slices);
    const int p0 = (rg.t_begin + tl) * K;
    int d = -1;
    if (lane < K) {
      d = (early && item == item0) ? d_first : __ldg(inv_l + p0 + lane);
      if (d >= 0) d -= rg.row0;
      if (perm && sl == 0 && d >= 0) perm[d] = p0 + lane;
    }
    const int4 *src = x + (size_t)tl * row_vec;
    const int v0 = sl * (32 * U) + lane;
    int4 r[U];
#pragma unroll
    for (int u = 0; u < U; u++)
      if (v0 + u * 32 < row_vec) r[u] = ld16_stream(src + v0 + u * 32);
    for (int k = 0; k < K; k++) {
      const int dk = __shfl_sync(0xffffffffu, d, k);
      if (dk < 0) continue;
      int4 *dst = buf + (size_t)dk * row_vec;
#pragma unroll
      for (int u = 0; u < U; u++)
        if (v0 + u * 32 < row_vec) st16_stream(dst + v0 + u * 32, r[u]);
    }
  }
}

#ifdef FOREMOE_TUNING   // the register-staged LSU combine: a sweep alternative, not selected by the product build
// =============================================================================================
// a6: combine.  y[t][h] = sum_k w[t][k] * float(eo[inv[t*K+k]][h]), fp32 fma, k ascending from
// acc = 0 (order / fma / fp32 output = DESIGN.md reading 16).
// One warp per (token, slice) item; per lane KB * U independent 16-byte loads in flight
// (k in groups of KB, masked tail), fma into registers, 16-byte stores of the fp32 row.
// =============================================================================================

template <bool kBf16, int KB, int U>
__global__ void __launch_bounds__(256)
k_combine_rows(const int32_t *__restrict__ inv_l, const float *__restrict__ w_l,
               const int32_t *__restrict__ mb_off, int mb_begin, int mb_end, int K, int row_vec,
               int n_slices, const int4 *__restrict__ eo, float4 *__restrict__ y) {
  constexpr int kF = kBf16 ? 8 : 4;          // floats produced per 16-byte input vector
  pdl_wait_then_release();
  const RangeInfo rg = load_range(mb_off, mb_begin, mb_end, K);
  const int lane = threadIdx.x & 31;
  const long long n_items = (long long)(rg.t_end - rg.t_begin) * n_slices;
  const long long warps = (long long)gridDim.x * (blockDim.x >> 5);
  for (long long item = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
       item < n_items; item += warps) {
    const int tl = (int)(item / n_slices);
    const int sl = (int)(item - (long long)tl * n_slices);
    const int p0 = (rg.t_begin + tl) * K;
    int d = -1;
    float wv = 0.f;
    if (lane < K) {
      d = __ldg(inv_l + p0 + lane);
      if (d >= 0) d -= rg.row0;
      wv = w_l ? __ldg(w_l + p0 + lane) : 1.f;     // w_l == nullptr: unit weights (dispatch backward)
    }
    const int v0 = sl * (32 * U) + lane;
    float acc[U][kF];
#pragma unroll
    for (int u = 0; u < U; u++)
#pragma unroll
      for (int f = 0; f < kF; f++) acc[u][f] = 0.f;

    for (int k0 = 0; k0 < K; k0 += KB) {
      int4 r[KB][U];
      float wk[KB];
      bool on[KB];
#pragma unroll
      for (int kk = 0; kk < KB; kk++) {
        const int k = k0 + kk;
        const int dk = __shfl_sync(0xffffffffu, d, k & 31);
        wk[kk] = __shfl_sync(0xffffffffu, wv, k & 31);
        on[kk] = (k < K) && (dk >= 0);
        const int4 *src = eo + (size_t)(on[kk] ? dk : 0) * row_vec;
#pragma unroll
        for (int u = 0; u < U; u++)
          if (on[kk] && v0 + u * 32 < row_vec) r[kk][u] = ld16_stream(src + v0 + u * 32);
      }
#pragma unroll
      for (int kk = 0; kk < KB; kk++) {
        if (!on[kk]) continue;
#pragma unroll
        for (int u = 0; u < U; u++) {
          if (kBf16) {
            acc[u][0] = __fmaf_rn(wk[kk], bf16_lo(r[kk][u].x), acc[u][0]);
            acc[u][1] = __fmaf_rn(wk[kk], bf16_hi(r[kk][u].x), acc[u][1]);
            acc[u][2] = __fmaf_rn(wk[kk], bf16_lo(r[kk][u].y), acc[u][2]);
            acc[u][3] = __fmaf_rn(wk[kk], bf16_hi(r[kk][u].y), acc[u][3]);
            acc[u][4] = __fmaf_rn(wk[kk], bf16_lo(r[kk][u].z), acc[u][4]);
            acc[u][5] = __fmaf_rn(wk[kk], bf16_hi(r[kk][u].z), acc[u][5]);
            acc[u][6] = __fmaf_rn(wk[kk], bf16_lo(r[kk][u].w), acc[u][6]);
            acc[u][7] = __fmaf_rn(wk[kk], bf16_hi(r[kk][u].w), acc[u][7]);
          } else {
            acc[u][0] = __fmaf_rn(wk[kk], __int_as_float(r[kk][u].x), acc[u][0]);
            acc[u][1] = __fmaf_rn(wk[kk], __int_as_float(r[kk][u].y), acc[u][1]);
            acc[u][2] = __fmaf_rn(wk[kk], __int_as_float(r[kk][u].z), acc[u][2]);
            acc[u][3] = __fmaf_rn(wk[kk], __int_as_float(r[kk][u].w), acc[u][3]);
          }
        }
      }
    }
    // fp32 row of token tl: row_vec * kF floats = row_vec * kF / 4 float4
    float4 *dst = y + (size_t)tl * row_vec * (kF / 4);
#pragma unroll
    for (int u = 0; u < U; u++) {
      const int v = v0 + u * 32;
      if (v < row_vec) {
        int4 o;
        o.x = __float_as_int(acc[u][0]); o.y = __float_as_int(acc[u][1]);
        o.z = __float_as_int(acc[u][2]); o.w = __float_as_int(acc[u][3]);
        st16_stream(dst + (size_t)v * (kF / 4), o);
        if (kBf16) {
          o.x = __float_as_int(acc[u][4]); o.y = __float_as_int(acc[u][5]);
          o.z = __float_as_int(acc[u][6]); o.w = __float_as_int(acc[u][7]);
          st16_stream(dst + (size_t)v * 2 + 1, o);
        }
      }
    }
  }
}

#endif  // FOREMOE_TUNING

// ---- launch configuration -------------------------------------------------------------------------
#ifdef FOREMOE_TUNING
DataTuning g_tune;
#endif

template <int U>
static int launch_dispatch(const Dims &d, const int32_t *inv_l, const int32_t *mb_off, int mb_begin,
                           int mb_end, const void *x, int32_t *perm, void *buf, cudaStream_t st,
                           bool prepare) {
  static DeviceMemo memo;
  const int occ = launch_facts(k_dispatch_rows<U>, memo, 256, 0);
  if (!occ) return FOREMOE_ERR_CUDA;
  if (prepare) return FOREMOE_OK;
  // Oversubscribed grid, about one (token, slice) item per warp although only `occ` CTAs are
  // resident per SM: the store path runs ~10 % faster with fresh CTAs streaming in than with a
  // strictly persistent grid (profiles/r01_sweeps.md).  The item count of a launch is estimated
  // from the mean micro-step of the shape (mb_off lives on the device): 4..128 CTAs per SM.
  const int n_slices = (d.row_vec + 32 * U - 1) / (32 * U);
  int per_sm = g_tune.dispatch_cta_per_sm;
  if (per_sm <= 0) {
    const long long items = (long long)(d.T / d.n_mb + 1) * n_slices;
    const long long want = (items + 8LL * num_sms() - 1) / (8LL * num_sms());
    per_sm = 4;
    while (per_sm < want && per_sm < 128) per_sm <<= 1;
    if (per_sm < occ) per_sm = occ;
  }
  const cudaError_t e = launch_pdl(k_dispatch_rows<U>, num_sms() * per_sm, 256, 0, st, inv_l, mb_off,
                                   mb_begin, mb_end, d.K, d.row_vec, n_slices, (const int4 *)x, perm,
                                   (int4 *)buf, d.plan_stable);
  return e == cudaSuccess ? FOREMOE_OK : FOREMOE_ERR_CUDA;
}

#ifdef FOREMOE_TUNING
template <bool kBf16, int KB, int U>
static int launch_combine(const Dims &d, const int32_t *inv_l, const float *w_l,
                          const int32_t *mb_off, int mb_begin, int mb_end, const void *eo, float *y,
                          cudaStream_t st, bool prepare) {
  static DeviceMemo memo;
  const int occ = launch_facts(k_combine_rows<kBf16, KB, U>, memo, 256, 0);
  if (!occ) return FOREMOE_ERR_CUDA;
  if (prepare) return FOREMOE_OK;
  const int per_sm = g_tune.combine_cta_per_sm > 0 ? g_tune.combine_cta_per_sm : occ;
  const int n_slices = (d.row_vec + 32 * U - 1) / (32 * U);
  const cudaError_t e = launch_pdl(k_combine_rows<kBf16, KB, U>, num_sms() * per_sm, 256, 0, st, inv_l,
                                   w_l, mb_off, mb_begin, mb_end, d.K, d.row_vec, n_slices,
                                   (const int4 *)eo, (float4 *)y);
  return e == cudaSuccess ? FOREMOE_OK : FOREMOE_ERR_CUDA;
}

template <bool kBf16, int KB>
static int launch_combine_u(int U, const Dims &d, const int32_t *inv_l, const float *w_l,
                            const int32_t *mb_off, int mb_begin, int mb_end, const void *eo,
                            float *y, cudaStream_t st, bool prepare) {
  if (U >= 2) return launch_combine<kBf16, KB, 2>(d, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
  return launch_combine<kBf16, KB, 1>(d, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
}

template <bool kBf16>
static int launch_combine_kb(int KB, int U, const Dims &d, const int32_t *inv_l, const float *w_l,
                             const int32_t *mb_off, int mb_begin, int mb_end, const void *eo,
                             float *y, cudaStream_t st, bool prepare) {
#define FOREMOE_KB_CASE(n) \
  case n: return launch_combine_u<kBf16, n>(U, d, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
  switch (KB) {
    FOREMOE_KB_CASE(1) FOREMOE_KB_CASE(2) FOREMOE_KB_CASE(3) FOREMOE_KB_CASE(4)
    FOREMOE_KB_CASE(5) FOREMOE_KB_CASE(6) FOREMOE_KB_CASE(7) FOREMOE_KB_CASE(8)
  }
#undef FOREMOE_KB_CASE
  return FOREMOE_ERR_INVALID_ARG;
}

#endif  // FOREMOE_TUNING

static int check_range(const Dims &d, int layer, int mb_begin, int mb_end) {
  if (layer < 0 || layer >= d.L || mb_begin < 0 || mb_end > d.n_mb || mb_begin > mb_end)
    return FOREMOE_ERR_INVALID_ARG;
  return FOREMOE_OK;
}

// a4 + a5: selects the kernel variant of the shape and launches it (prepare: memoises its launch
// facts instead)
int dispatch_rows(const Dims &d, const int32_t *inv_l, const int32_t *mb_off, int mb_begin,
                  int mb_end, const void *x, int32_t *perm, void *buf, cudaStream_t st, bool prepare) {
  // auto: the bulk-copy ring wins from 8 KB rows on (config 5's 8 KB rows: 447 vs 457 us per launch, config 3's
  // 14 KB rows: 324 vs 327 us; profiles/r02_sweeps.md); at 4 KB the register-staged kernel is faster (97 vs 101 us)
  if (g_tune.dispatch_impl == 1 || (g_tune.dispatch_impl < 0 && d.row_bytes >= 8 * 1024)) {
    const int rc = launch_dispatch_tma(d, inv_l, mb_off, mb_begin, mb_end, x, perm, buf, st, prepare);
    if (rc != FOREMOE_ERR_INVALID_ARG) return rc;     // rows too large for the ring: fall through
  }
  int U = g_tune.dispatch_u;
  if (U <= 0) U = d.row_vec >= 64 ? 2 : 1;      // 1 KB slices: best or within 1 % of best on every config (sweep)
#ifdef FOREMOE_TUNING      // the auto rule above picks 1 or 2: wider slices exist for sweeps only
  if (U >= 8) return launch_dispatch<8>(d, inv_l, mb_off, mb_begin, mb_end, x, perm, buf, st, prepare);
  if (U >= 4) return launch_dispatch<4>(d, inv_l, mb_off, mb_begin, mb_end, x, perm, buf, st, prepare);
#endif
  if (U >= 2) return launch_dispatch<2>(d, inv_l, mb_off, mb_begin, mb_end, x, perm, buf, st, prepare);
  return launch_dispatch<1>(d, inv_l, mb_off, mb_begin, mb_end, x, perm, buf, st, prepare);
}

// a6 and its unit-weight form (w_l == nullptr sums the K rows: fma(1, v, acc) = acc + v exactly)
int combine_rows(const Dims &d, const int32_t *inv_l, const float *w_l, const int32_t *mb_off,
                 int mb_begin, int mb_end, const void *eo, float *y, cudaStream_t st, bool prepare) {
#ifndef FOREMOE_TUNING
  // The bulk-copy ring stages 512-byte slices, so it fits every legal shape (K = 32: 2 warps x 2 stages of
  // 32 x 512 B = 66 KB) and is the only combine kernel in the product library.
  return launch_combine_bulk(d, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
#else
  int rc;
  if (g_tune.combine_impl < 0 || g_tune.combine_impl == 2) {   // default: bulk-copy ring
    rc = launch_combine_bulk(d, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
    if (rc != FOREMOE_ERR_INVALID_ARG) return rc;
  }
  if (g_tune.combine_impl != 0) {    // cp.async ring
    rc = launch_combine_async(d, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
    if (rc != FOREMOE_ERR_INVALID_ARG) return rc;
  }
  const int groups = (d.K + 7) / 8;
  const int KB = (d.K + groups - 1) / groups;
  int U = g_tune.combine_u;
  if (U <= 0) U = (d.row_vec >= 64 && KB <= 4) ? 2 : 1;
  if (d.act_dtype == FOREMOE_ACT_BF16)
    return launch_combine_kb<true>(KB, U, d, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
  return launch_combine_kb<false>(KB, U, d, inv_l, w_l, mb_off, mb_begin, mb_end, eo, y, st, prepare);
#endif
}

}  // namespace foremoe

using namespace foremoe;

#ifdef FOREMOE_TUNING
// sweep builds only (not declared in include/foremoe.h): key = field index of DataTuning in
// declaration order
extern "C" __attribute__((visibility("default"))) void foremoe_tuning_set(int key, int value) {
  int *f[] = {&g_tune.dispatch_impl, &g_tune.dispatch_u, &g_tune.dispatch_cta_per_sm,
              &g_tune.dispatch_stages, &g_tune.dispatch_warps, &g_tune.combine_impl,
              &g_tune.combine_u, &g_tune.combine_cta_per_sm, &g_tune.combine_depth,
              &g_tune.combine_threads, &g_tune.pdl, &g_tune.bwd_depth, &g_tune.bwd_cta_per_sm,
              &g_tune.bwd_impl, &g_tune.hist_variant};
  if (key >= 0 && key < (int)(sizeof(f) / sizeof(f[0]))) *f[key] = value;
}
#endif

extern "C" __attribute__((visibility("default"))) int foremoe_dispatch(const foremoe_shape_t *shape, int32_t layer, int32_t mb_begin,
                                int32_t mb_end, const int32_t *mb_off, const int32_t *inv,
                                const void *x, int32_t *perm, void *buf, int32_t *dev_status,
                                void *stream) {
  (void)dev_status;
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if ((rc = check_range(d, layer, mb_begin, mb_end))) return rc;
  if (d.T == 0) return FOREMOE_OK;                     // a step without tokens: the plan arrays may be NULL
  if (!mb_off || !inv || !x || !buf || !aligned(x, 16) || !aligned(buf, 16))
    return FOREMOE_ERR_INVALID_ARG;
  if (mb_begin == mb_end) return FOREMOE_OK;
  return dispatch_rows(d, inv + (size_t)layer * d.T * d.K, mb_off, mb_begin, mb_end, x, perm, buf,
                       (cudaStream_t)stream, false);
}

static int combine_entry(const foremoe_shape_t *shape, int32_t layer, int32_t mb_begin,
                         int32_t mb_end, const int32_t *mb_off, const int32_t *inv, const float *w,
                         const void *expert_out, float *y, void *stream) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if ((rc = check_range(d, layer, mb_begin, mb_end))) return rc;
  if (d.T == 0) return FOREMOE_OK;
  if (!mb_off || !inv || !expert_out || !y || !aligned(expert_out, 16) || !aligned(y, 16))
    return FOREMOE_ERR_INVALID_ARG;
  if (mb_begin == mb_end) return FOREMOE_OK;
  const size_t lo = (size_t)layer * d.T * d.K;
  return combine_rows(d, inv + lo, w ? w + lo : nullptr, mb_off, mb_begin, mb_end, expert_out, y,
                      (cudaStream_t)stream, false);
}

extern "C" __attribute__((visibility("default"))) int foremoe_combine(const foremoe_shape_t *shape, int32_t layer, int32_t mb_begin,
                               int32_t mb_end, const int32_t *mb_off, const int32_t *inv,
                               const float *w, const void *expert_out, float *y,
                               int32_t *dev_status, void *stream) {
  (void)dev_status;
  if (!w && !(shape && shape->T == 0)) return FOREMOE_ERR_INVALID_ARG;
  return combine_entry(shape, layer, mb_begin, mb_end, mb_off, inv, w, expert_out, y, stream);
}

extern "C" __attribute__((visibility("default"))) int foremoe_dispatch_bwd(const foremoe_shape_t *shape, int32_t layer, int32_t mb_begin,
                                    int32_t mb_end, const int32_t *mb_off, const int32_t *inv,
                                    const void *d_buf, float *dx, int32_t *dev_status, void *stream) {
  (void)dev_status;
  return combine_entry(shape, layer, mb_begin, mb_end, mb_off, inv, nullptr, d_buf, dx, stream);
}

// Memoises the launch facts (occupancy, shared-memory opt-in) of every data-path kernel variant this
// shape selects, on the calling thread's current device: after it the data-path calls make no CUDA
// call other than the launch, so they can be stream-captured from the first call on.
extern "C" __attribute__((visibility("default"))) int foremoe_warmup(const foremoe_shape_t *shape, void *stream) {
  (void)stream;
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  if ((rc = dispatch_rows(d, nullptr, nullptr, 0, 0, nullptr, nullptr, nullptr, nullptr, true))) return rc;
  if ((rc = combine_rows(d, nullptr, nullptr, nullptr, 0, 0, nullptr, nullptr, nullptr, true))) return rc;
  if ((rc = combine_bwd_rows(d, nullptr, nullptr, nullptr, 0, 0, nullptr, nullptr, nullptr, nullptr, nullptr, true, true))) return rc;
  if ((rc = combine_bwd_rows(d, nullptr, nullptr, nullptr, 0, 0, nullptr, nullptr, nullptr, nullptr, nullptr, false, true))) return rc;
  num_sms();
  return FOREMOE_OK;
}

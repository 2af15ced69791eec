// Dispatch (a4 + a5) with the TMA bulk-copy engine: the row of token t is pulled ONCE into shared
// memory with cp.async.bulk (global -> shared, completion on an mbarrier) and pushed to its K
// destination rows with K cp.async.bulk (shared -> global) copies -- no register staging, one
// instruction per 4-14 KB row, so the LSU store queue is out of the picture.
// Each warp runs its own ring of `NS` row-sized stages; nothing is shared between warps.
#include "foremoe_data.cuh"

namespace foremoe {

// smem layout: [warps][NS][row_bytes] rows (16-byte aligned), then [warps][NS] mbarriers (8 B),
// then [warps][NS][32] destination rows.
__global__ void __launch_bounds__(512)
k_dispatch_tma(const int32_t *__restrict__ inv_l, const int32_t *__restrict__ mb_off, int mb_begin,
               int mb_end, int K, int row_bytes, int NS, const char *__restrict__ x,
               int32_t *__restrict__ perm, char *__restrict__ buf, int early) {
  extern __shared__ __align__(128) unsigned char smem[];
  if (!early) pdl_wait_then_release();
  const int n_warps = blockDim.x >> 5;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  unsigned char *rows = smem + (size_t)warp * NS * row_bytes;
  uint64_t *bars = (uint64_t *)(smem + (size_t)n_warps * NS * row_bytes) + warp * NS;
  int32_t *dbuf = (int32_t *)(smem + (size_t)n_warps * NS * row_bytes + (size_t)n_warps * NS * 8) +
                  (size_t)warp * NS * 32;
  const RangeInfo rg = load_range(mb_off, mb_begin, mb_end, K);
  if (early) pdl_wait_then_release();      // only mb_off was read (FOREMOE_FLAG_PLAN_STABLE)
  const int n_tok = rg.t_end - rg.t_begin;
  const int W = gridDim.x * n_warps;
  const int w0 = blockIdx.x * n_warps + warp;
  const int n_my = w0 < n_tok ? (n_tok - w0 + W - 1) / W : 0;

  if (lane == 0)
    for (int s = 0; s < NS; s++) mbar_init(smem_u32(bars + s), 1);
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  __syncwarp();

  // producer side of item n (token w0 + n*W) into stage n % NS
  auto load_item = [&](int n) {
    const int s = n % NS;
    const int tl = w0 + n * W;
    if (lane < K) dbuf[s * 32 + lane] = __ldg(inv_l + (size_t)(rg.t_begin + tl) * K + lane);
    if (lane == 0) {
      const uint32_t bar = smem_u32(bars + s);
      mbar_expect_tx(bar, (uint32_t)row_bytes);
      bulk_g2s(smem_u32(rows + (size_t)s * row_bytes), x + (size_t)tl * row_bytes, (uint32_t)row_bytes, bar);
    }
  };

  // the stage of item j-2 is refilled in iteration j: its stores had one iteration to drain
  const int ahead = NS - 2;
  for (int n = 0; n < ahead && n < n_my; n++) load_item(n);
  for (int j = 0; j < n_my; j++) {
    if (lane < K) bulk_wait_read<1>();     // stores of item j-2 have left shared memory
    __syncwarp();
    if (j + ahead < n_my) load_item(j + ahead);
    const int s = j % NS;
    mbar_wait(smem_u32(bars + s), (uint32_t)((j / NS) & 1));
    if (lane < K) {
      int d = dbuf[s * 32 + lane];
      if (d >= 0) {
        d -= rg.row0;
        bulk_s2g(buf + (size_t)d * row_bytes, smem_u32(rows + (size_t)s * row_bytes), (uint32_t)row_bytes);
        if (perm) perm[d] = (rg.t_begin + w0 + j * W) * K + lane;
      }
      bulk_commit();
    }
  }
  if (lane < K) bulk_wait_all();
}

int launch_dispatch_tma(const Dims &d, const int32_t *inv_l, const int32_t *mb_off, int mb_begin,
                        int mb_end, const void *x, int32_t *perm, void *buf, cudaStream_t st,
                        bool prepare) {
  const size_t budget = 200 * 1024;
  int warps = g_tune.dispatch_warps > 0 ? g_tune.dispatch_warps : (d.row_bytes <= 4096 ? 8 : 4);
  if (warps > 16) warps = 16;
  const size_t per_stage = (size_t)d.row_bytes + 8 + 128;
  int NS = g_tune.dispatch_stages > 0 ? g_tune.dispatch_stages : (int)(budget / (per_stage * warps));
  if (NS > 8) NS = 8;
  while (NS >= 3 && per_stage * warps * NS > budget) NS--;
  if (NS < 3) return FOREMOE_ERR_INVALID_ARG;       // rows too large for a ring: caller falls back
  const size_t smem = per_stage * warps * NS;
  static DeviceMemo memo;
  if (!launch_facts(k_dispatch_tma, memo, warps * 32, smem)) return FOREMOE_ERR_CUDA;
  if (prepare) return FOREMOE_OK;
  const int per_sm = g_tune.dispatch_cta_per_sm > 0 ? g_tune.dispatch_cta_per_sm : 14;   // sweep: r02_sweeps.md
  const cudaError_t e = launch_pdl(k_dispatch_tma, num_sms() * per_sm, warps * 32, smem, st, inv_l, mb_off,
                                   mb_begin, mb_end, d.K, d.row_bytes, NS, (const char *)x, perm, (char *)buf,
                                   d.plan_stable);
  return e == cudaSuccess ? FOREMOE_OK : FOREMOE_ERR_CUDA;
}

}  // namespace foremoe

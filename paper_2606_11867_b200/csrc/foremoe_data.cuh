// Internal: helpers shared by the data-path kernels (dispatch / combine) and their launchers.
#pragma once

#include "foremoe_common.cuh"

namespace foremoe {

// Launch parameters of the data path.  In the product build they are compile-time defaults (chosen
// from the ncu evidence under profiles/) and nothing can change them; a sweep build
// (python -m paper_2606_11867_b200.build --tuning: -DFOREMOE_TUNING, a separate libforemoe_tuning.so)
// makes them mutable through foremoe_tuning_set, which is not part of include/foremoe.h.
struct DataTuning {
  int dispatch_impl = -1;        // -1 auto, 0 = register-staged LSU rows, 1 = TMA bulk-copy ring
  int dispatch_u = 0;            // impl 0: 16-byte vectors per lane per item (0 = auto)
  int dispatch_cta_per_sm = 0;   // 0 = auto
  int dispatch_stages = 0;       // impl 1: ring stages per warp (0 = auto)
  int dispatch_warps = 0;        // impl 1: warps per CTA (0 = auto)
  int combine_impl = -1;         // -1 auto, 0 = register-staged LSU rows, 1 = cp.async ring, 2 = bulk-copy ring
  int combine_u = 0;             // impl 0 / 2: 16-byte vectors per lane per row slice (0 = auto)
  int combine_cta_per_sm = 0;
  int combine_depth = 0;         // impl 1 / 2: stages in flight (0 = auto)
  int combine_threads = 0;       // impl 1 / 2: threads per CTA (0 = auto)
  int pdl = 1;                   // programmatic dependent launch on the data-path kernels
  int bwd_depth = 0;             // k_combine_bwd: stages in flight per thread (0 = auto)
  int bwd_cta_per_sm = 0;        // 0 = auto
  int bwd_impl = -1;             // reserved: k_combine_bwd has one implementation (cp.async ring); the value is ignored
  int hist_variant = 2;          // k_load_hist: 0 = 4-byte loads, 1 = warp-aggregated, 2 = 16-byte loads
};
#ifdef FOREMOE_TUNING
extern DataTuning g_tune;
#else
constexpr DataTuning g_tune{};
#endif

struct RangeInfo { int t_begin, t_end, row0; };

__device__ __forceinline__ RangeInfo load_range(const int32_t *__restrict__ mb_off, int mb_begin,
                                                int mb_end, int K) {
  RangeInfo r;
  r.t_begin = __ldg(mb_off + mb_begin);
  r.t_end = __ldg(mb_off + mb_end);
  r.row0 = r.t_begin * K;
  return r;
}

// rows of x / expert_out are read once per launch and rows of buf / y are written once: keep them
// out of L1 and mark them streaming.
__device__ __forceinline__ int4 ld16_stream(const void *p) {
  int4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0, %1, %2, %3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}
__device__ __forceinline__ void st16_stream(void *p, const int4 &v) {
  asm volatile("st.global.cs.v4.s32 [%0], {%1, %2, %3, %4};"
               :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

__device__ __forceinline__ float bf16_lo(int v) { return __int_as_float(v << 16); }
__device__ __forceinline__ float bf16_hi(int v) { return __int_as_float(v & 0xffff0000); }

__device__ __forceinline__ uint32_t smem_u32(const void *p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}

// 16-byte asynchronous global -> shared copies (LDGSTS) and their group fences: the shared-memory
// rings of k_combine_async / k_combine_bwd
__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" :: "n"(N) : "memory"); }

// Programmatic dependent launch: the kernel may be scheduled while the previous kernel of the
// stream drains (hides launch latency and the ramp).  The predecessor's writes are only guaranteed
// visible after pdl_wait(), whether or not it triggers early, so a kernel touches no global memory
// before it -- except the plan arrays (mb_off, inv, w) when the caller set FOREMOE_FLAG_PLAN_STABLE
// (`early`): then the first plan entries are fetched while the predecessor drains.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
// Every PDL kernel of the library releases its own dependents only AFTER its own wait has returned.
// A dependent can then become resident no earlier than the completion of this kernel's predecessor,
// and so on down the stream: whatever a chain of library kernels overlaps, it never overlaps a kernel
// launched before the chain's first member.  This is what lets a FOREMOE_FLAG_PLAN_STABLE kernel fetch
// plan entries ahead of its wait when only the kernel launched immediately before it is known not to
// write them -- [writer of w] -> dispatch -> combine(PLAN_STABLE) would otherwise let the combine read
// w while the writer runs (the dispatch, still waiting on the writer, would already have released it).
__device__ __forceinline__ void pdl_wait_then_release() { pdl_wait(); pdl_launch_dependents(); }

template <typename... KArgs, typename... Args>
static cudaError_t launch_pdl(void (*kern)(KArgs...), int grid, int block, size_t smem, cudaStream_t st,
                              Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)block);
  cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = g_tune.pdl ? 1 : 0;
  cfg.attrs = attr; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

template <typename Kern>
static int occupancy_ctas(Kern kern, int threads, size_t smem = 0) {
  int n = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, threads, smem) != cudaSuccess || n <= 0) n = 1;
  return n;
}

constexpr int kSmemOptIn = 227 * 1024;   // largest dynamic shared memory a CTA can opt into on sm_100a

// Resident CTAs per SM (>= 1) of `kern` at (threads, smem) on the calling thread's current device,
// memoised per device in `memo` (one DeviceMemo per kernel instantiation).  On a miss the kernel is
// opted into the full shared-memory carve-out (always the same value, so shapes with different
// footprints cannot undo each other) and the occupancy is queried: neither is allowed during stream
// capture, which is what foremoe_warmup is for.  Returns 0 on a CUDA error.
template <typename Kern>
static int launch_facts(Kern kern, DeviceMemo &memo, int threads, size_t smem) {
  const int dev = current_device();
  const uint64_t key = (uint64_t)smem * 2048 + (uint64_t)threads;
  int occ = memo.get(dev, key);
  if (occ) return occ;
  if (smem > 48 * 1024 &&
      cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemOptIn) != cudaSuccess)
    return 0;
  occ = occupancy_ctas(kern, threads, smem);
  memo.put(dev, key, occ);
  return occ;
}

// Every launcher takes `prepare`: true = memoise the launch facts of the variant this shape selects
// and return without launching (foremoe_warmup).
// launchers of the ring variants; return FOREMOE_ERR_INVALID_ARG when the shape does not fit the
// variant (the caller then uses the next one)
int launch_dispatch_tma(const Dims &d, const int32_t *inv_l, const int32_t *mb_off, int mb_begin,
                        int mb_end, const void *x, int32_t *perm, void *buf, cudaStream_t st,
                        bool prepare);
int launch_combine_async(const Dims &d, const int32_t *inv_l, const float *w_l,
                         const int32_t *mb_off, int mb_begin, int mb_end, const void *eo, float *y,
                         cudaStream_t st, bool prepare);
int launch_combine_bulk(const Dims &d, const int32_t *inv_l, const float *w_l,
                        const int32_t *mb_off, int mb_begin, int mb_end, const void *eo, float *y,
                        cudaStream_t st, bool prepare);

// backward of a6 (foremoe_backward.cu): want_dw selects the variant that also reads expert_out
int combine_bwd_rows(const Dims &d, const int32_t *inv_l, const float *w_l, const int32_t *mb_off,
                     int mb_begin, int mb_end, const float *dy, const void *eo, void *d_eo, float *dw_l,
                     cudaStream_t st, bool want_dw, bool prepare);

// mbarrier + bulk-copy (TMA, 1-D) primitives shared by the bulk rings
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}"
      :: "r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               :: "r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void *dst, uint32_t src, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
               :: "l"(dst), "r"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() {
  asm volatile("cp.async.bulk.wait_group.read %0;" :: "n"(N) : "memory");
}
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
// orders generic-proxy accesses to shared memory before later async-proxy (bulk-copy) accesses
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

}  // namespace foremoe

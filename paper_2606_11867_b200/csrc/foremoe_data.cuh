// Internal: helpers shared by the data-path kernels (dispatch / combine) and their launchers.
#pragma once

#include "foremoe_common.cuh"

namespace foremoe {

// Tunables of the data path (defaults chosen from the ncu evidence under profiles/; the debug
// setter exists for sweeps only).
struct DataTuning {
  int dispatch_impl = -1;        // -1 auto, 0 = register-staged LSU rows, 1 = TMA bulk-copy ring
  int dispatch_u = 0;            // impl 0: 16-byte vectors per lane per item (0 = auto)
  int dispatch_cta_per_sm = 0;   // 0 = occupancy
  int dispatch_stages = 0;       // impl 1: ring stages per warp (0 = auto)
  int dispatch_warps = 0;        // impl 1: warps per CTA (0 = auto)
  int combine_impl = -1;         // -1 auto, 0 = register-staged LSU rows, 1 = cp.async smem ring
  int combine_u = 0;             // impl 0
  int combine_cta_per_sm = 0;
  int combine_depth = 0;         // impl 1: stages in flight per thread (0 = auto)
  int combine_threads = 0;       // impl 1: threads per CTA (0 = auto)
  int pdl = 1;                   // programmatic dependent launch on the data-path kernels
  int bwd_depth = 0;             // k_combine_bwd: stages in flight per thread (0 = auto)
  int bwd_cta_per_sm = 0;        // 0 = occupancy
};
extern DataTuning g_tune;

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
// stream drains (hides launch latency and the ramp); it touches no global memory before pdl_wait():
// the predecessor's writes are only guaranteed visible after the wait, whether or not it triggers early.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

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

// launchers of the asynchronous variants; return FOREMOE_ERR_INVALID_ARG when the shape does not
// fit the variant (the caller then uses the register-staged kernel)
int launch_dispatch_tma(const Dims &d, const int32_t *inv_l, const int32_t *mb_off, int mb_begin,
                        int mb_end, const void *x, int32_t *perm, void *buf, cudaStream_t st);
int launch_combine_async(const Dims &d, const int32_t *inv_l, const float *w_l,
                         const int32_t *mb_off, int mb_begin, int mb_end, const void *eo, float *y,
                         cudaStream_t st);

}  // namespace foremoe

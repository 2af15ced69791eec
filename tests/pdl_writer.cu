// Test fixture only (built by tests/test_gpu_pdl_chain.py with nvcc; not part of the library).
// A deliberately slow writer that behaves like a caller's own PDL-aware kernel: it releases its
// dependents at once, spins for `spin_cycles` clocks, and only then copies src -> dst.  A kernel
// launched behind it with programmatic stream serialisation is resident while the copy is pending.
#include <cuda_runtime.h>
#include <stdint.h>

__global__ void k_slow_copy(const float *__restrict__ src, float *__restrict__ dst, long long n,
                            long long spin_cycles) {
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const long long t0 = clock64();
  while (clock64() - t0 < spin_cycles) {}
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
    dst[i] = src[i];
}

extern "C" int slow_copy(const float *src, float *dst, long long n, long long spin_cycles, void *stream) {
  k_slow_copy<<<2, 256, 0, (cudaStream_t)stream>>>(src, dst, n, spin_cycles);
  return (int)cudaGetLastError();
}

// pic_check.cuh — index checks of the debug build (-DPIC_BOUNDS_CHECK=1, libpic_b200_check.so).
// compute-sanitizer is closed on the GPU pool this was developed on, so the kernels carry their
// own bounds checks: every shared- and global-memory index that is computed from particle data
// (cell indices, sort keys, scatter destinations, queue positions) goes through chk(i, n).  In
// the production build chk is the identity and costs nothing; in the check build an index outside
// [0, n) is counted in g_bounds_violations (read by pic_debug_bounds) and replaced by 0, so that
// the run continues and the count is what the tests see (tests/test_gpu_bounds_check.py).
#pragma once
#include <cuda_runtime.h>

#ifndef PIC_BOUNDS_CHECK
#define PIC_BOUNDS_CHECK 0
#endif

namespace picb200 {
#if PIC_BOUNDS_CHECK
extern __device__ unsigned long long g_bounds_violations;   // defined in pic_api.cu (-rdc=true)
template <typename I>
__device__ __forceinline__ I chk(I i, long long n) {
  if ((long long)i < 0 || (long long)i >= n) {
    atomicAdd(&g_bounds_violations, 1ull);
    return (I)0;
  }
  return i;
}
#else
template <typename I>
__device__ __forceinline__ I chk(I i, long long) { return i; }
#endif
}  // namespace picb200

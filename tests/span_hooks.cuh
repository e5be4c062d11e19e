// Test infrastructure, NOT part of the product: force-included (nvcc -include) into a second build of
// greenlantern_b200.cu by tests/test_gpu_parity.py::test_device_span_of_one_step.  It fills hot_kernel's
// no-op phase hook GLH_TL(k) (gl_hot.cuh) with two %globaltimer stamps -- the start of a CTA's first unit
// (k = 0: minimum over the grid) and the moment a chi^2 has been written (k = 5: maximum over the grid) --
// and exports gl_debug_span to read them.  The difference is the ON-DEVICE span of one launch, which CUDA
// events cannot resolve on this hardware (they see the end of a kernel on a 2.048-us grid: bench.py,
// roofline.event_time_vs_kernel_time).
#pragma once
#include <cuda_runtime.h>
__device__ unsigned long long g_span[2] = {~0ull, 0ull};
__device__ __forceinline__ unsigned long long glh_gtime() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
#define GLH_TL(k)                                                                   \
    do {                                                                            \
        if ((k) == 0 && threadIdx.x == 0) atomicMin(&g_span[0], glh_gtime());       \
        if ((k) == 5 && threadIdx.x == 0) atomicMax(&g_span[1], glh_gtime());       \
    } while (0)
// out[0], out[1] = first start, last end [ns of the GPU's global timer]; reset != 0 re-arms the stamps
extern "C" int gl_debug_span(unsigned long long* out, int reset) {
    cudaError_t e = cudaMemcpyFromSymbol(out, g_span, 16);
    if (e == cudaSuccess && reset) {
        unsigned long long z[2] = {~0ull, 0ull};
        e = cudaMemcpyToSymbol(g_span, z, 16);
    }
    return e == cudaSuccess ? 0 : -2;
}

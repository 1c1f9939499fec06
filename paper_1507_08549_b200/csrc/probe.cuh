// probe.cuh -- the roofline denominator of the L2-bound configurations, measured by the library itself.
// MEASURED_PEAKS.json holds the HBM copy bandwidth only; SURVEY.md section 8(d) asks for the L2 peak to be measured on
// the box ("L2-resident read / copy").  Two plain kernels over a working set that stays in the 126 MB L2: a copy
// (read + write bytes, the figure bench.py uses as `roofline.peak` for the L2-bound rows) and a read-only pass
// (`peak_read`).  Not part of the solve path.
#pragma once
#include "common.cuh"

namespace snp {

constexpr int kProbeThreads = 1024;

// b[i] = a[i] for `reps` passes; grid-stride, 4 independent 16-byte accesses in flight per thread, L1 bypassed.
__global__ void __launch_bounds__(kProbeThreads) k_probe_l2_copy(const double2* __restrict__ a, double2* __restrict__ b,
                                                                size_t n2, int reps) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (int r = 0; r < reps; ++r) {
        size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
        for (; i + 3 * stride < n2; i += 4 * stride) {
            const double2 v0 = __ldcg(a + i), v1 = __ldcg(a + i + stride), v2 = __ldcg(a + i + 2 * stride),
                          v3 = __ldcg(a + i + 3 * stride);
            __stcg(b + i, v0); __stcg(b + i + stride, v1); __stcg(b + i + 2 * stride, v2); __stcg(b + i + 3 * stride, v3);
        }
        for (; i < n2; i += stride) __stcg(b + i, __ldcg(a + i));
    }
}

// sum of a[] for `reps` passes (the sum keeps the loads alive; one store per thread at the end).
__global__ void __launch_bounds__(kProbeThreads) k_probe_l2_read(const double2* __restrict__ a, size_t n2, int reps,
                                                                double* __restrict__ sink) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    double s0 = 0, s1 = 0, s2 = 0, s3 = 0;
    for (int r = 0; r < reps; ++r) {
        size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
        for (; i + 3 * stride < n2; i += 4 * stride) {
            const double2 v0 = __ldcg(a + i), v1 = __ldcg(a + i + stride), v2 = __ldcg(a + i + 2 * stride),
                          v3 = __ldcg(a + i + 3 * stride);
            s0 += v0.x + v0.y; s1 += v1.x + v1.y; s2 += v2.x + v2.y; s3 += v3.x + v3.y;
        }
        for (; i < n2; i += stride) { const double2 v = __ldcg(a + i); s0 += v.x + v.y; }
    }
    sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = (s0 + s1) + (s2 + s3);
}

}  // namespace snp

// tiling.h -- tile / box geometry of the resident kernel, shared by the host planner and the device code so that
// both derive the same numbers.  Plain C++ (no CUDA types): also compiled by g++ in tests/test_tiling.py, which
// brute-forces the coverage property below on the CPU.
//
// One axis of n cells is cut into nt owned intervals [t*own, min(n,(t+1)*own)); own is a multiple of the patch
// alignment q (4 cells in r, H cells in z).  The CTA of tile t works on a box of B cells starting at
// box_origin(); the box must contain the owned interval widened by the margin h = 2m on every side that has a
// neighbour (clipped to [0,n)), because m red-black sweeps move the domain of dependence by 2m cells
// (DESIGN.md §6).
#pragma once

#ifdef __CUDACC__
#define SNP_HD __host__ __device__ __forceinline__
#else
#define SNP_HD inline
#endif

namespace snp {

// Origin of the box of the tile whose owned interval starts at x0: x0 - h rounded down to the alignment q, clamped
// so that the box [origin, origin + B) stays inside [0, n).  Requires n % q == 0, B % q == 0, n >= B.
SNP_HD int box_origin(int x0, int h, int q, int B, int n) {
    int o = x0 - h;
    if (o < 0) o = 0;
    o = (o / q) * q;
    if (o > n - B) o = n - B;
    return o;
}

// Cells lost at the low side by rounding x0 - h down to a multiple of q (x0 is a multiple of q).
SNP_HD int origin_slack(int h, int q) { return (q - h % q) % q; }

// Tiling of one axis.  Returns false if a box of B cells cannot hold one aligned tile plus its margins.
SNP_HD bool plan_axis(int n, int B, int h, int q, int* nt, int* own) {
    if (n % q != 0 || B % q != 0 || n < B) return false;
    if (n == B) {
        *nt = 1;
        *own = n;
        return true;
    }
    const int omax = ((B - 2 * h - origin_slack(h, q)) / q) * q;
    if (omax < q) return false;
    int t = (n + omax - 1) / omax;
    int o = (((n + t - 1) / t + q - 1) / q) * q;     // balanced, rounded up to q
    if (o > omax) o = omax;
    t = (n + o - 1) / o;
    *nt = t;
    *own = o;
    return true;
}

// The property the kernel relies on, for tile t.
SNP_HD bool box_covers(int t, int own, int h, int q, int B, int n) {
    const int x0 = t * own;
    const int x1 = x0 + own < n ? x0 + own : n;
    const int lo = x0 - h > 0 ? x0 - h : 0;
    const int hi = x1 + h < n ? x1 + h : n;
    const int o = box_origin(x0, h, q, B, n);
    return o >= 0 && o % q == 0 && o + B <= n && o <= lo && o + B >= hi;
}

}  // namespace snp

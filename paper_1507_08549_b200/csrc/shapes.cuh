// shapes.cuh -- the instantiations of the on-chip sweep kernels (resident: sweep_resident.cuh, blocked:
// sweep_blocked.cuh) as a table of launchable shapes.  Every shape is instantiated in its own translation unit
// (shape_tu.cu compiled once per -DSNP_TU=<n>) so that the library builds in parallel; sn_poisson.cu only sees the
// tables.  Host-side metadata only: no arithmetic of the method lives here.
#pragma once
#include <cstddef>

namespace snp {

struct ShapeInfo {
    int H, TXN, TYN, minb;
    size_t smem, smem_ring, smem_ring_ds;
    const void* fn[5];          // [0] block mode, [1] halo mode, [2] halo mode inside one cluster (DSMEM) or NULL,
                                // [3] halo mode with ring duty, [4] cluster halo mode with ring duty or NULL
    int BW() const { return 4 * TXN; }
    int BH() const { return H * TYN; }
    int NT() const { return TXN * TYN; }
    int threads() const { return TXN * TYN + 32; }     // + the service warp
    size_t smem_of(int f) const { return f == 3 ? smem_ring : f == 4 ? smem_ring_ds : smem; }
};

struct BlkShapeInfo {
    int H, TXN, TYN, minb;
    size_t smem;
    const void* fn;
    double hs_clk;             // measured clocks per half-sweep of one box with `minb` CTAs sharing an SM (cost model)
    int BW() const { return 4 * TXN; }
    int BH() const { return H * TYN; }
    int NT() const { return TXN * TYN; }
};

constexpr int kNumResShapes = 11, kNumBlkShapes = 5;
// defined in shape_tu.cu (one translation unit per resident shape, one for all blocked shapes)
ShapeInfo res_shape(int i);
BlkShapeInfo blk_shape(int i);
template <int I> ShapeInfo res_shape_tu();
BlkShapeInfo blk_shape_tu(int i);

}  // namespace snp

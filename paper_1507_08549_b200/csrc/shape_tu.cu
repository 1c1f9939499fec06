// shape_tu.cu -- compiled once per -DSNP_TU=<n>: n = 0 .. kNumResShapes-1 instantiates the resident kernels of shape n
// (block mode, halo mode, ring duty, and the cluster / DSMEM variants where the shape supports them), n = 100 the
// blocked kernels, n = 200 the dispatch by index.  See shapes.cuh.
#include "shapes.cuh"

#ifndef SNP_TU
#error "compile with -DSNP_TU=<n>"
#endif

#if SNP_TU < 100
#include "sweep_resident.cuh"
namespace snp {
namespace {
template <int H, int TXN, int TYN, int MINB, bool DS = true, bool HALO = true>
ShapeInfo shape_of() {
    const void *ds = nullptr, *dsr = nullptr;
    if constexpr (!HALO) {
        return {H, TXN, TYN, MINB, ResShape<H, TXN, TYN>::smem_bytes, 0, 0,
                {(const void*)k_sor_resident<H, TXN, TYN, MINB, false, false>, nullptr, nullptr, nullptr, nullptr}};
    } else {
    if constexpr (DS) {
        ds = (const void*)k_sor_resident<H, TXN, TYN, MINB, true, false, true>;
        dsr = (const void*)k_sor_resident<H, TXN, TYN, MINB, true, true, true>;
    }
    return {H, TXN, TYN, MINB, ResShape<H, TXN, TYN>::smem_bytes, ResShape<H, TXN, TYN>::smem_bytes_ring,
            ResShape<H, TXN, TYN>::smem_bytes_ring_ds,
            {(const void*)k_sor_resident<H, TXN, TYN, MINB, false, false>,
             (const void*)k_sor_resident<H, TXN, TYN, MINB, true, false>, ds,
             (const void*)k_sor_resident<H, TXN, TYN, MINB, true, true>, dsr}};
    }
}
}  // namespace
template <>
ShapeInfo res_shape_tu<SNP_TU>() {
#if SNP_TU == 0
    return shape_of<8, 32, 14, 1, false>();   // box 128 x 112, 448 threads
#elif SNP_TU == 1
    return shape_of<8, 32, 8, 1, false>();    // box 128 x 64,  256 threads
#elif SNP_TU == 2
    return shape_of<8, 16, 8, 2>();           // box 64 x 64,   128 threads
#elif SNP_TU == 3
    return shape_of<4, 16, 8, 2>();           // box 64 x 32,   128 threads
#elif SNP_TU == 4
    return shape_of<4, 8, 8, 2>();            // box 32 x 32,    64 threads
#elif SNP_TU == 5
    return shape_of<2, 8, 16, 2>();           // box 32 x 32,   128 threads
#elif SNP_TU == 6
    return shape_of<8, 32, 7, 2, false>();    // box 128 x 56,  224 threads, 2 CTAs / SM (halo mode on chip-filling grids)
#elif SNP_TU == 7
    return shape_of<4, 16, 16, 1>();          // box 64 x 64,   256 threads
#elif SNP_TU == 8
    return shape_of<6, 12, 8, 2>();           // box 48 x 48,    96 threads
#elif SNP_TU == 9
    return shape_of<4, 12, 16, 1>();          // box 48 x 64,   192 threads
#elif SNP_TU == 10
    return shape_of<2, 16, 32, 1>();          // box 64 x 64,   512 threads of 2 x 4 patches (shortest half-sweep: small grids)
#else
#error "unknown resident shape"
#endif
}
}  // namespace snp

#elif SNP_TU == 100
#include "sweep_blocked.cuh"
namespace snp {
namespace {
template <int H, int TXN, int TYN, int MINB>
BlkShapeInfo blk_shape_of(double hs_clk) {
    return {H, TXN, TYN, MINB, BlkShape<H, TXN, TYN>::smem_bytes, (const void*)k_sor_blocked<H, TXN, TYN, MINB>, hs_clk};
}
}  // namespace
BlkShapeInfo blk_shape_tu(int i) {
    switch (i) {
        case 0: return blk_shape_of<8, 32, 8, 2>(1853.0);     // box 128 x 64,  256 threads, 2 CTAs / SM
        case 1: return blk_shape_of<8, 32, 14, 1>(1516.0);    // box 128 x 112, 448 threads
        case 2: return blk_shape_of<16, 32, 8, 1>(1562.0);    // box 128 x 128, 256 threads
        case 3: return blk_shape_of<8, 16, 8, 3>(1400.0);     // box 64 x 64,   128 threads, 3 CTAs / SM
        default: return blk_shape_of<4, 16, 8, 4>(1200.0);    // box 64 x 32,   128 threads, 4 CTAs / SM
    }
}
}  // namespace snp

#else   // SNP_TU == 200: dispatch by index
namespace snp {
template <> ShapeInfo res_shape_tu<0>();
template <> ShapeInfo res_shape_tu<1>();
template <> ShapeInfo res_shape_tu<2>();
template <> ShapeInfo res_shape_tu<3>();
template <> ShapeInfo res_shape_tu<4>();
template <> ShapeInfo res_shape_tu<5>();
template <> ShapeInfo res_shape_tu<6>();
template <> ShapeInfo res_shape_tu<7>();
template <> ShapeInfo res_shape_tu<8>();
template <> ShapeInfo res_shape_tu<9>();
template <> ShapeInfo res_shape_tu<10>();
ShapeInfo res_shape(int i) {
    switch (i) {
        case 0: return res_shape_tu<0>();
        case 1: return res_shape_tu<1>();
        case 2: return res_shape_tu<2>();
        case 3: return res_shape_tu<3>();
        case 4: return res_shape_tu<4>();
        case 5: return res_shape_tu<5>();
        case 6: return res_shape_tu<6>();
        case 7: return res_shape_tu<7>();
        case 8: return res_shape_tu<8>();
        case 9: return res_shape_tu<9>();
        default: return res_shape_tu<10>();
    }
}
BlkShapeInfo blk_shape(int i) { return blk_shape_tu(i); }
}  // namespace snp
#endif

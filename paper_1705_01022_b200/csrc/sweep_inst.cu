// Instantiations of the sweep kernels.  Compiled once per (family, log2 D):
//     -DOCT_INST_FAMILY=0 -DOCT_INST_LOG2D=5|6|7|8     bit-packed kernel (sweep.cuh)
//     -DOCT_INST_FAMILY=1 -DOCT_INST_LOG2D=5|6|7|8     link-entry kernel (sweep_links.cuh)
// (paper_1705_01022_b200/build.py runs the compilations in parallel and links them with oct_api.cu).
#include "launch.h"
#include "sweep.cuh"
#include "sweep_links.cuh"

#define OCT_CAT2(a, b) a##b
#define OCT_CAT(a, b) OCT_CAT2(a, b)

namespace octb {

#if OCT_INST_FAMILY == 0
// ---- bit-packed kernel: (log2 D, tcx, tcy) combinations the library is built for ---------------------
#ifndef OCT_CELLS_PER_WARP
#define OCT_CELLS_PER_WARP 128   // cells carried by one warp (4 per lane; 8 overflows the instruction cache, profiles/r1_a)
#endif
constexpr int pick_wpd(int log2d, int tcx, int tcy)
{
    const int ncell = ((1 << log2d) / (4 << tcx)) * ((1 << log2d) / (4 << tcy));
    return ncell <= OCT_CELLS_PER_WARP ? 1 : ncell / OCT_CELLS_PER_WARP;
}

template <int LD, int TX, int TY, int BLK>
SweepLaunch make_launch()
{
    constexpr int W = pick_wpd(LD, TX, TY);
    using SH = SweepShape<LD, TX, TY, W>;
    return SweepLaunch{sweep_kernel<LD, TX, TY, BLK, W>, nullptr, SH::NTHREADS, SH::SMEM_BYTES, SH::DPB};
}

#define OCT_SHAPES_5(X) X(5, 0, 0) X(5, 1, 1) X(5, 2, 2)
#define OCT_SHAPES_6(X) X(6, 0, 0) X(6, 1, 1) X(6, 2, 2) X(6, 2, 1) X(6, 3, 1) X(6, 1, 3)
#define OCT_SHAPES_7(X) X(7, 0, 0) X(7, 1, 1) X(7, 2, 2) X(7, 2, 1) X(7, 3, 2) X(7, 4, 1) X(7, 3, 1) X(7, 1, 3)
#define OCT_SHAPES_8(X) X(8, 1, 1) X(8, 2, 2) X(8, 2, 1) X(8, 3, 2) X(8, 4, 1)

bool OCT_CAT(oct_find_packed_, OCT_INST_LOG2D)(int tx, int ty, int blk, SweepLaunch* out)
{
#define X(LD, TX, TY)                                                               \
    if (tx == TX && ty == TY) {                                                     \
        if (blk == kBlkSync) { *out = make_launch<LD, TX, TY, kBlkSync>(); return true; }       \
        if (blk == kBlkDelayed) { *out = make_launch<LD, TX, TY, kBlkDelayed>(); return true; } \
        if constexpr (TX >= 1 && TY >= 1) {                                         \
            if (blk == kBlkDT) { *out = make_launch<LD, TX, TY, kBlkDT>(); return true; }       \
        }                                                                           \
        return false;                                                               \
    }
    OCT_CAT(OCT_SHAPES_, OCT_INST_LOG2D)(X)
#undef X
    return false;
}

#else
// ---- link-entry kernel: (log2 D, tcx, tcy, threads per domain, domains per CTA, bytes per entry) ----------
// Variant A is the default (the faster one on B200: D = 64 TC=1,1 one warp per domain, two cells per lane,
// warp-level synchronisation only, four-byte entries; shapes with few cells per domain -- TC=2,2 (half a warp per 64 x 64
// domain), TC=3,2 and TC=4,1 -- two-byte entries, which double the domains in flight: measured per shape, profiles/r2_sweep.md;
// D = 128 TC=1,1 four warps with two cells per lane), variant B the alternative work split or entry size of the shapes the
// paper's results rest on.  BATCH (many lattices per launch) is built for the
// small-lattice shapes (D <= 64, and D = 128 TC=1,1: BASELINE config 2 runs its ensembles at L = 1024 with D = 128), where one
// lattice cannot fill the GPU.
template <int LD, int TX, int TY, int BLK, int G, int DPB, int EB>
SweepLaunch make_links_launch(bool dead)
{
    using SH = LinkShape<LD, TX, TY, G, DPB, EB>;
    SweepLaunch sl{dead ? sweep_links_kernel<LD, TX, TY, BLK, G, DPB, true, false, EB> : sweep_links_kernel<LD, TX, TY, BLK, G, DPB, false, false, EB>,
                   nullptr, SH::NTHREADS, SH::SMEM_BYTES, SH::DPB};
    if constexpr (LD <= 6 || (LD == 7 && TX == 1 && TY == 1))
        sl.kern_batch = dead ? sweep_links_kernel<LD, TX, TY, BLK, G, DPB, true, true, EB> : sweep_links_kernel<LD, TX, TY, BLK, G, DPB, false, true, EB>;
    return sl;
}

#define OCT_LINK_SHAPES_A_5(X) X(5, 0, 0, 32, 4, 4) X(5, 1, 1, 16, 8, 4)
#define OCT_LINK_SHAPES_A_6(X) X(6, 0, 0, 128, 1, 4) X(6, 1, 1, 32, 4, 4) X(6, 2, 1, 32, 4, 4) X(6, 2, 2, 16, 4, 2) X(6, 3, 1, 16, 4, 2) X(6, 1, 3, 16, 4, 2)
#define OCT_LINK_SHAPES_A_7(X) X(7, 0, 0, 256, 1, 4) X(7, 1, 1, 128, 1, 4) X(7, 2, 2, 64, 1, 2) X(7, 2, 1, 128, 1, 4) X(7, 3, 2, 32, 1, 2) X(7, 4, 1, 32, 1, 2) X(7, 3, 1, 64, 1, 2) X(7, 1, 3, 64, 1, 2)
#define OCT_LINK_SHAPES_A_8(X) X(8, 1, 1, 512, 1, 2) X(8, 2, 1, 512, 1, 2) X(8, 2, 2, 256, 1, 2) X(8, 3, 2, 128, 1, 2) X(8, 4, 1, 128, 1, 2)
#define OCT_LINK_SHAPES_B_5(X)
#define OCT_LINK_SHAPES_B_6(X) X(6, 1, 1, 64, 2, 4) X(6, 2, 2, 16, 2, 4)
#define OCT_LINK_SHAPES_B_7(X) X(7, 1, 1, 256, 1, 4) X(7, 2, 2, 64, 1, 4)
#define OCT_LINK_SHAPES_B_8(X) X(8, 1, 1, 1024, 1, 2)

bool OCT_CAT(oct_find_links_, OCT_INST_LOG2D)(int tx, int ty, int blk, bool variant_b, bool dead, SweepLaunch* out)
{
#define X(LD, TX, TY, G, DPB, EB)                                                                    \
    if (tx == TX && ty == TY) {                                                                      \
        if (blk == kBlkSync) { *out = make_links_launch<LD, TX, TY, kBlkSync, G, DPB, EB>(dead); return true; }       \
        if (blk == kBlkDelayed) { *out = make_links_launch<LD, TX, TY, kBlkDelayed, G, DPB, EB>(dead); return true; } \
        if constexpr (TX >= 1 && TY >= 1) {                                                          \
            if (blk == kBlkDT) { *out = make_links_launch<LD, TX, TY, kBlkDT, G, DPB, EB>(dead); return true; }       \
        }                                                                                            \
        return false;                                                                                \
    }
    if (variant_b) { OCT_CAT(OCT_LINK_SHAPES_B_, OCT_INST_LOG2D)(X) }
    OCT_CAT(OCT_LINK_SHAPES_A_, OCT_INST_LOG2D)(X)
#undef X
    return false;
}
#endif

}  // namespace octb

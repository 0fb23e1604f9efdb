// Host-side dispatch between oct_api.cu and the translation units that instantiate the sweep kernels
// (sweep_inst.cu is compiled once per kernel family and domain size, so that the library builds in parallel).
#pragma once
#include "sweep.cuh"

namespace octb {

struct SweepLaunch {
    void (*kern)(const SweepParams);
    void (*kern_batch)(const SweepBatchParams);   // nullptr: this shape has no many-lattices-per-launch variant
    int threads, smem, dpb;
};

// bit-packed kernel (sweep.cuh), domains of 2^ld sites; false if (tx, ty, blk) is not built
bool oct_find_packed_5(int tx, int ty, int blk, SweepLaunch* out);
bool oct_find_packed_6(int tx, int ty, int blk, SweepLaunch* out);
bool oct_find_packed_7(int tx, int ty, int blk, SweepLaunch* out);
bool oct_find_packed_8(int tx, int ty, int blk, SweepLaunch* out);
// link-entry kernel (sweep_links.cuh); variant_b: the alternative work split where one is built
bool oct_find_links_5(int tx, int ty, int blk, bool variant_b, bool dead, SweepLaunch* out);
bool oct_find_links_6(int tx, int ty, int blk, bool variant_b, bool dead, SweepLaunch* out);
bool oct_find_links_7(int tx, int ty, int blk, bool variant_b, bool dead, SweepLaunch* out);
bool oct_find_links_8(int tx, int ty, int blk, bool variant_b, bool dead, SweepLaunch* out);   // D = 256: two-byte entries only

}  // namespace octb

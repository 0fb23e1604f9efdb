// Height reconstruction and the integer reductions for W^2(t) and C_h(t,s).
//
// Heights are the discrete integral of the slopes (the slope field is curl-free), so
//   h(x,y) - h(0,0) = sum_{j=1..y} sigma_y(0,j) + sum_{i=1..x} sigma_x(i,y).
// Kernel 1 (column_gather_kernel + column_anchor_kernel, here) scans column 0 once: anchor[y] = h(0,y) - h(0,0).
// Kernel 2 (observe_rows.cuh) gives every warp one word-row (4 site rows, L/4 packed words) and either
// stores the heights or accumulates the centred sums.  One pass over the packed lattice, no
// intermediate arrays.  This header also holds the parameter block and the small utility kernels.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace octb {

// ---- kernel 1: anchor[y] = sum_{j=1..y} sigma_y(0,j) -----------------------------------------------------
// sigma_y(0, 4wy+j) is bit 8j+1 of word (wx=0, wy).  Column 0 is strided by one lattice row per word: L/4 separate
// 32-byte sectors.  One SM cannot keep enough of them in flight (a single CTA doing the strided reads and the scan took
// 25 us at L = 2^16, a tenth of the W^2 pass it precedes; profiles/r2_observables.md), so the pass is two grids of CTAs of
// kColThreads words each: column_gather_kernel copies the column into a compact array and leaves every CTA's net slope
// in blocksum[]; column_anchor_kernel scans its own words and adds the sums of the CTAs before it.
constexpr int kColThreads = 256;
constexpr int kColMaxBlocks = 128;     // L <= 2^17: 2^15 words in column 0

__device__ __forceinline__ int word_dy(uint32_t v) { return 2 * __popc(v & 0x02020202u) - 4; }   // net sigma_y of the word's first column

__device__ __forceinline__ void column_gather_body(const uint32_t* __restrict__ lat, uint32_t L, uint32_t* __restrict__ col,
                                                   int32_t* __restrict__ blocksum)
{
    __shared__ int32_t wsum[kColThreads / 32];
    const uint32_t LW = L >> 2;
    const uint32_t w = blockIdx.x * kColThreads + threadIdx.x;
    int s = 0;
    if (w < LW) {
        const uint32_t v = lat[(size_t)w * LW];
        col[w] = v;
        s = word_dy(v);
    }
    s = __reduce_add_sync(0xFFFFFFFFu, s);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        int t = 0;
#pragma unroll
        for (int k = 0; k < kColThreads / 32; ++k) t += wsum[k];
        blocksum[blockIdx.x] = t;
    }
}

// anchors of the words of CTA blockIdx.x; also clears the n_zero output words of the reduction that follows (this kernel
// precedes it in the stream: no separate memset)
__device__ __forceinline__ void column_anchor_body(const uint32_t* __restrict__ col, const int32_t* __restrict__ blocksum, uint32_t L,
                                                   int32_t* __restrict__ anchor, unsigned long long* __restrict__ zero, int n_zero)
{
    __shared__ int32_t wtot[kColThreads / 32];
    __shared__ int32_t base;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (blockIdx.x == 0 && (int)threadIdx.x < n_zero) zero[threadIdx.x] = 0ull;
    const uint32_t LW = L >> 2;
    const uint32_t w = blockIdx.x * kColThreads + threadIdx.x;
    const uint32_t v = w < LW ? col[w] : 0x02020000u;                 // zero net slope past the end
    const int s = word_dy(v);
    int incl = s;                                                     // inclusive scan inside the warp
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const int u = __shfl_up_sync(0xFFFFFFFFu, incl, off);
        if (lane >= off) incl += u;
    }
    if (lane == 31) wtot[warp] = incl;
    if (warp == 0) {
        // net slope of the CTAs before this one.  The scan counts sigma_y(0,0) as well, which closes the loop around the
        // torus and is not part of the path from (0,0); remove it.
        int t = 0;
#pragma unroll
        for (int k = 0; k < kColMaxBlocks / 32; ++k) {
            const uint32_t bidx = (uint32_t)(lane + 32 * k);
            if (bidx < blockIdx.x) t += blocksum[bidx];
        }
        t = __reduce_add_sync(0xFFFFFFFFu, t);
        if (lane == 0) base = t - ((col[0] >> 1) & 1u ? 1 : -1);
    }
    __syncthreads();
    int run = base + incl - s;                                        // value entering this thread's word
    for (int k = 0; k < warp; ++k) run += wtot[k];
    if (w < LW) {
        int32_t a[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            run += (v >> (8 * j + 1)) & 1u ? 1 : -1;
            a[j] = run;
        }
        *reinterpret_cast<int4*>(anchor + 4 * w) = make_int4(a[0], a[1], a[2], a[3]);
    }
}

// A second translation unit that only wants the device bodies and parameter blocks of this header (width2_static.cu)
// defines OCT_OBSERVE_BODIES_ONLY: the non-template kernels below have external linkage and must exist once per library.
#ifndef OCT_OBSERVE_BODIES_ONLY
// the lattices k = blockIdx.y (one or two: current lattice and snapshot)
__global__ void __launch_bounds__(kColThreads)
column_gather_kernel(const uint32_t* __restrict__ lat0, const uint32_t* __restrict__ lat1, uint32_t L,
                     uint32_t* __restrict__ col0, uint32_t* __restrict__ col1, int32_t* __restrict__ blocksum)
{
    column_gather_body(blockIdx.y ? lat1 : lat0, L, blockIdx.y ? col1 : col0, blocksum + blockIdx.y * kColMaxBlocks);
}

__global__ void __launch_bounds__(kColThreads)
column_anchor_kernel(const uint32_t* __restrict__ col0, const uint32_t* __restrict__ col1, const int32_t* __restrict__ blocksum, uint32_t L,
                     int32_t* __restrict__ anchor0, int32_t* __restrict__ anchor1, unsigned long long* __restrict__ zero, int n_zero)
{
    column_anchor_body(blockIdx.y ? col1 : col0, blocksum + blockIdx.y * kColMaxBlocks, L, blockIdx.y ? anchor1 : anchor0, zero,
                       blockIdx.y ? 0 : n_zero);
}

#endif  // OCT_OBSERVE_BODIES_ONLY

// ---- kernel 2 -------------------------------------------------------------------------------------

struct RowsParams {
    const uint32_t* latA;        // current lattice
    const uint32_t* latB;        // snapshot (autocorr) or nullptr
    const int32_t* anchorA;      // h(0,y) - h(0,0) for latA
    const int32_t* anchorB;
    const unsigned long long* countersA;    // [0] net, [1] h00 of the current lattice
    const long long* snapB;                 // {h00, net} of the snapshot
    int32_t* heights;                       // heights_kernel output
    unsigned long long* out;                // rows3_kernel: [0..3] W^2 sums, [4..8] C_h sums, [9..14] C_s sums
    unsigned long long* out_ch;             // where the five C_h sums go: out + 4 in the 16-slot layout, the caller's buffer itself for oct_autocorr
    uint32_t L;
};

// ---- the same for an ensemble (oct_observe_batch): one launch covers the members blockIdx.z / .y ---------------------
constexpr int kMaxObsBatch = 64;
struct ObsMember {
    const uint32_t* latA;
    const uint32_t* latB;                   // snapshot or nullptr
    int32_t* anchorA;
    int32_t* anchorB;
    uint32_t* colA;
    uint32_t* colB;
    int32_t* blocksum;                      // 2 x kColMaxBlocks
    const unsigned long long* countersA;
    const long long* snapB;
    unsigned long long* out;                // 16 int64 of this member
};
struct ObsBatchParams {
    uint32_t L;
    int n_zero;
    ObsMember m[kMaxObsBatch];
};

#ifndef OCT_OBSERVE_BODIES_ONLY
__global__ void __launch_bounds__(kColThreads) column_gather_batch_kernel(const __grid_constant__ ObsBatchParams BP)
{
    const ObsMember& mb = BP.m[blockIdx.z];
    column_gather_body(blockIdx.y ? mb.latB : mb.latA, BP.L, blockIdx.y ? mb.colB : mb.colA, mb.blocksum + blockIdx.y * kColMaxBlocks);
}

__global__ void __launch_bounds__(kColThreads) column_anchor_batch_kernel(const __grid_constant__ ObsBatchParams BP)
{
    const ObsMember& mb = BP.m[blockIdx.z];
    column_anchor_body(blockIdx.y ? mb.colB : mb.colA, mb.blocksum + blockIdx.y * kColMaxBlocks, BP.L, blockIdx.y ? mb.anchorB : mb.anchorA,
                       mb.out, blockIdx.y ? 0 : BP.n_zero);
}

// ---- slope (lattice-gas) autocorrelation C_s(t,s), PAPER.md:85-88 --------------------------------------
// n = slope bit.  out = {sum nx_t nx_s, sum ny_t ny_s, sum nx_t, sum ny_t, sum nx_s, sum ny_s}: one streaming
// pass over both packed lattices (0.5 B/site), six POPC per word pair, grid-stride, int64 atomics per CTA.
constexpr int kSlopeThreads = 256;

__global__ void __launch_bounds__(kSlopeThreads)
slope_autocorr_kernel(const uint4* __restrict__ A, const uint4* __restrict__ B, size_t n_vec, unsigned long long* __restrict__ out)
{
    constexpr uint32_t MX = 0x55555555u, MY = 0xAAAAAAAAu;
    unsigned int c[6] = {0, 0, 0, 0, 0, 0};      // per thread: < 2^32 bits even at L = 2^17 with >= 2^10 threads
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_vec; i += (size_t)gridDim.x * blockDim.x) {
        const uint4 a = A[i], b = B[i];
        const uint32_t aw[4] = {a.x, a.y, a.z, a.w}, bw[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uint32_t ab = aw[k] & bw[k];
            c[0] += __popc(ab & MX); c[1] += __popc(ab & MY);
            c[2] += __popc(aw[k] & MX); c[3] += __popc(aw[k] & MY);
            c[4] += __popc(bw[k] & MX); c[5] += __popc(bw[k] & MY);
        }
    }
    __shared__ unsigned long long red[6][kSlopeThreads / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const unsigned int v = __reduce_add_sync(0xFFFFFFFFu, c[k]);      // a warp's total stays far below 2^32
        if (lane == 0) red[k][warp] = v;
    }
    __syncthreads();
    if (threadIdx.x < 6) {
        unsigned long long t = 0;
        for (int w = 0; w < kSlopeThreads / 32; ++w) t += red[threadIdx.x][w];
        atomicAdd(&out[threadIdx.x], t);
    }
}

// ---- init ------------------------------------------------------------------------------------------
__global__ void fill_words_kernel(uint4* __restrict__ lat, size_t n_vec, uint32_t word)
{
    const uint4 v = make_uint4(word, word, word, word);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_vec; i += (size_t)gridDim.x * blockDim.x) lat[i] = v;
}

__global__ void snapshot_anchor_kernel(const unsigned long long* counters, long long* out)
{
    out[0] = (long long)counters[1];   // h(0,0)
    out[1] = (long long)counters[0];   // net
}

__global__ void set_counters_kernel(unsigned long long* counters, long long h00, long long net)
{
    counters[0] = (unsigned long long)net;
    counters[1] = (unsigned long long)h00;
}

#endif  // OCT_OBSERVE_BODIES_ONLY

}  // namespace octb

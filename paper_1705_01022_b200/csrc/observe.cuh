// Height reconstruction and the integer reductions for W^2(t) and C_h(t,s).
//
// Heights are the discrete integral of the slopes (the slope field is curl-free), so
//   h(x,y) - h(0,0) = sum_{j=1..y} sigma_y(0,j) + sum_{i=1..x} sigma_x(i,y).
// Kernel 1 (column_anchor_kernel) scans column 0 once: anchor[y] = h(0,y) - h(0,0).
// Kernel 2 (rows_kernel) gives every warp one word-row (4 site rows, L/4 packed words): the warp
// streams the row 128 bytes at a time, turns each word's four sigma_x nibbles into row increments,
// shuffle-scans them across the lanes, carries the running height in registers and either stores
// the 16 heights of its word (coalesced 16-byte stores) or accumulates the centred sums.  One pass
// over the packed lattice, no intermediate arrays.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace octb {

// ---- kernel 1: anchor[y] = sum_{j=1..y} sigma_y(0,j), one CTA ---------------------------------------
// sigma_y(0, 4wy+j) is bit 8j+1 of word (wx=0, wy).
constexpr int kAnchorThreads = 1024;

__global__ void __launch_bounds__(kAnchorThreads)
column_anchor_kernel(const uint32_t* __restrict__ lat, uint32_t L, int32_t* __restrict__ anchor)
{
    __shared__ int32_t part[kAnchorThreads];
    const uint32_t LW = L >> 2;
    const uint32_t per = (LW + kAnchorThreads - 1) / kAnchorThreads;     // words of column 0 per thread
    const uint32_t w0 = threadIdx.x * per;
    int32_t sum = 0;
    for (uint32_t w = w0; w < w0 + per && w < LW; ++w) {
        const uint32_t v = lat[(size_t)w * LW];
        sum += 2 * __popc(v & 0x02020202u) - 4;
    }
    part[threadIdx.x] = sum;
    __syncthreads();
    // inclusive Hillis-Steele scan over the per-thread totals
    for (int off = 1; off < kAnchorThreads; off <<= 1) {
        int32_t v = threadIdx.x >= (unsigned)off ? part[threadIdx.x - off] : 0;
        __syncthreads();
        part[threadIdx.x] += v;
        __syncthreads();
    }
    // h(0, 4*w0 - 1 + 1 ...) : running value entering this thread's first word.  The scan counts
    // sigma_y(0,0) as well, which closes the loop around the torus and is not part of the path from
    // (0,0); remove it.
    const int32_t s00 = (lat[0] >> 1) & 1u ? 1 : -1;
    int32_t run = part[threadIdx.x] - sum - s00;
    for (uint32_t w = w0; w < w0 + per && w < LW; ++w) {
        const uint32_t v = lat[(size_t)w * LW];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            run += (v >> (8 * j + 1)) & 1u ? 1 : -1;
            anchor[4 * w + j] = run;
        }
    }
}

// ---- kernel 2 -------------------------------------------------------------------------------------
enum : int { kModeHeights = 0, kModeWidth2 = 1, kModeAutocorr = 2 };
constexpr int kRowsWarps = 8;

struct RowsParams {
    const uint32_t* latA;        // current lattice
    const uint32_t* latB;        // snapshot (autocorr) or nullptr
    const int32_t* anchorA;      // h(0,y) - h(0,0) for latA
    const int32_t* anchorB;
    const unsigned long long* countersA;    // [0] net, [1] h00 of the current lattice
    const long long* snapB;                 // {h00, net} of the snapshot
    int32_t* heights;                       // kModeHeights output
    unsigned long long* out;                // kModeWidth2: {S1,S2,c,net}; kModeAutocorr: {St,Ss,Sts,ct,cs}
    uint32_t L;
};

// Row increments of one packed word: r_j = (#up - #down) of the four sigma_x bits of sub-row j,
// biased to 0..8 (2*popc) and packed as four 16-bit fields so one 64-bit scan serves all four rows.
__device__ __forceinline__ unsigned long long packed_row_sums(uint32_t w)
{
    const uint32_t a = 2u * __popc(w & 0x00000055u), b = 2u * __popc(w & 0x00005500u);
    const uint32_t c = 2u * __popc(w & 0x00550000u), d = 2u * __popc(w & 0x55000000u);
    return (unsigned long long)(a | (b << 16)) | ((unsigned long long)(c | (d << 16)) << 32);
}

__device__ __forceinline__ unsigned long long warp_inclusive_scan(unsigned long long v, int lane)
{
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const unsigned long long u = __shfl_up_sync(0xFFFFFFFFu, v, off);
        if (lane >= off) v += u;
    }
    return v;
}

// One lattice stream of a warp: running (relative) heights at the left edge of the current chunk.
struct RowStream {
    const uint32_t* row;     // first word of this word-row
    int32_t left[4];         // h(4*wx0 - 1, 4*wy + j) - h(0,0) for the chunk starting at word wx0

    __device__ __forceinline__ void init(const uint32_t* lat, const int32_t* anchor, uint32_t LW, uint32_t wy)
    {
        row = lat + (size_t)wy * LW;
        const uint32_t w0 = row[0];
#pragma unroll
        for (int j = 0; j < 4; ++j)   // h(-1,y) = h(0,y) - sigma_x(0,y)
            left[j] = anchor[4 * wy + j] - ((w0 >> (8 * j)) & 1u ? 1 : -1);
    }

    // heights (relative to h00) of the 16 sites of this lane's word of the chunk: e[j][i]
    __device__ __forceinline__ void chunk(uint32_t w, int lane, int32_t (&e)[4][4])
    {
        const unsigned long long incl = warp_inclusive_scan(packed_row_sums(w), lane);
        const unsigned long long excl = incl - packed_row_sums(w);
        const unsigned long long tot = __shfl_sync(0xFFFFFFFFu, incl, 31);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            // un-bias: each preceding word contributed +4 per row
            int32_t h = left[j] + (int32_t)((excl >> (16 * j)) & 0xFFFFu) - 4 * lane;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                h += (w >> (8 * j + 2 * i)) & 1u ? 1 : -1;
                e[j][i] = h;
            }
            left[j] += (int32_t)((tot >> (16 * j)) & 0xFFFFu) - 4 * 32;
        }
    }
};

template <int MODE>
__global__ void __launch_bounds__(kRowsWarps * 32) rows_kernel(const RowsParams P)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t LW = P.L >> 2;
    const uint32_t wy = blockIdx.x * kRowsWarps + warp;     // word-row of this warp
    long long s1 = 0, s2 = 0, s3 = 0;

    if (wy < LW) {
        RowStream A, B;
        A.init(P.latA, P.anchorA, LW, wy);
        if constexpr (MODE == kModeAutocorr) B.init(P.latB, P.anchorB, LW, wy);
        const int32_t h00 = MODE == kModeHeights ? (int32_t)(long long)P.countersA[1] : 0;

        // L >= 16 => LW >= 4; chunks of 32 words, the last (only) chunk may be ragged when LW < 32
        for (uint32_t wx0 = 0; wx0 < LW; wx0 += 32) {
            const uint32_t wx = wx0 + lane;
            const bool ok = wx < LW;
            // a missing word must contribute zero increments: 0x..55 pattern has popc 2 per row -> r=0
            const uint32_t wa = ok ? A.row[wx] : 0x05050505u;
            int32_t ea[4][4];
            A.chunk(wa, lane, ea);
            if constexpr (MODE == kModeHeights) {
                if (ok) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        int4 v = make_int4(ea[j][0] + h00, ea[j][1] + h00, ea[j][2] + h00, ea[j][3] + h00);
                        *reinterpret_cast<int4*>(P.heights + (size_t)(4 * wy + j) * P.L + 4 * wx) = v;
                    }
                }
            } else if constexpr (MODE == kModeWidth2) {
                if (ok) {
#pragma unroll
                    for (int j = 0; j < 4; ++j)
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            s1 += ea[j][i];
                            s2 += (long long)ea[j][i] * ea[j][i];
                        }
                }
            } else {
                const uint32_t wb = ok ? B.row[wx] : 0x05050505u;
                int32_t eb[4][4];
                B.chunk(wb, lane, eb);
                if (ok) {
#pragma unroll
                    for (int j = 0; j < 4; ++j)
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            s1 += ea[j][i];
                            s2 += eb[j][i];
                            s3 += (long long)ea[j][i] * eb[j][i];
                        }
                }
            }
        }
    }

    if constexpr (MODE != kModeHeights) {
        __shared__ long long red[3][kRowsWarps];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            s1 += __shfl_xor_sync(0xFFFFFFFFu, s1, off);
            s2 += __shfl_xor_sync(0xFFFFFFFFu, s2, off);
            if constexpr (MODE == kModeAutocorr) s3 += __shfl_xor_sync(0xFFFFFFFFu, s3, off);
        }
        if (lane == 0) { red[0][warp] = s1; red[1][warp] = s2; red[2][warp] = s3; }
        __syncthreads();
        if (threadIdx.x == 0) {
            long long t1 = 0, t2 = 0, t3 = 0;
            for (int w = 0; w < kRowsWarps; ++w) { t1 += red[0][w]; t2 += red[1][w]; t3 += red[2][w]; }
            atomicAdd(&P.out[0], (unsigned long long)t1);
            atomicAdd(&P.out[1], (unsigned long long)t2);
            if constexpr (MODE == kModeAutocorr) atomicAdd(&P.out[2], (unsigned long long)t3);
            if (blockIdx.x == 0) {
                if constexpr (MODE == kModeWidth2) {
                    P.out[2] = P.countersA[1];             // c = h(0,0)
                    P.out[3] = P.countersA[0];             // net
                } else {
                    P.out[3] = P.countersA[1];             // c_t
                    P.out[4] = (unsigned long long)P.snapB[0];   // c_s
                }
            }
        }
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

}  // namespace octb

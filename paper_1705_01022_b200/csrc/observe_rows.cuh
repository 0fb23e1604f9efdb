// Row-streaming kernels for height reconstruction (a8) and the W^2 / C_h reductions (a9), second version.
//
// One warp owns one word-row (4 site rows, L/4 packed words).  Per chunk every lane takes RUN
// *consecutive* words (RUN/4 coalesced 128-bit loads; the warp reads 128*RUN contiguous bytes), walks
// them in registers and only then the warp does ONE shuffle scan to place the lanes' runs one after the
// other -- instead of a 64-bit scan per word as in the first version (profiles/r1_a: 554 GB/s).
//
// Inside a word the four site rows are handled byte-parallel: byte j of a register belongs to site row
// 4*wy + j.  With P_i = number of up-links among the first i sites of the row (bytewise prefix sums of
// the sigma_x bits) the height of site (i, j) of the word is
//       e_ij = left_j + 2 P_ij - i ,      left_j = height just west of the word in row j.
// Reductions: over a lane's run of <= 64 sites every height stays within +-73 of the height s at the start
// of the run (rows of one word differ by at most 5 there), so the heights are carried ENTIRELY in unsigned
// bytes,  H_i = base + 2 P_i - i * 0x01010101  with  base_j = left_j - s + 128,  and sum H, sum H^2 (or
// sum H_A H_B) are plain DP4A accumulations; the bias and s come off once per run in int64:
//       sum (s + r)^2 = n s^2 + 2 s sum r + sum r^2 .
// base needs no scan: at the first word of a run its row differences are read off the sigma_y bits of
// that word's first column (curl-freeness), and it advances by 2 P_4 - 4 per word.
// Heights: the same bytes relative to a 32-bit running height r0 (RowRun / word_heights below).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "observe.cuh"

namespace octb {

constexpr uint32_t kOnes = 0x01010101u;

// running state of one lattice stream inside a lane's run
struct RowRun {
    int r0;          // left_0 - 16, relative to the height at the start of the run
    uint32_t dq;     // bytes d_j + 16
};

// bytewise prefix counts of the sigma_x bits of a word: P[i-1] byte j = #up-links among sites 0..i-1 of row j
__device__ __forceinline__ void prefix_counts(uint32_t w, uint32_t (&P)[4])
{
    P[0] = w & kOnes;
    P[1] = P[0] + ((w >> 2) & kOnes);
    P[2] = P[1] + ((w >> 4) & kOnes);
    P[3] = P[2] + ((w >> 6) & kOnes);
}

// H_i bytes (heights of the word's sites minus r0) and the advance of the run state to the next word
__device__ __forceinline__ void word_heights(uint32_t w, RowRun& st, uint32_t (&H)[4], int& r0_here)
{
    uint32_t P[4];
    prefix_counts(w, P);
#pragma unroll
    for (int i = 0; i < 4; ++i) H[i] = st.dq - (uint32_t)(i + 1) * kOnes + 2u * P[i];
    r0_here = st.r0;
    const uint32_t t0 = P[3] & 0xFFu;
    st.r0 += 2 * (int)t0 - 4;
    st.dq = st.dq + 2u * P[3] - 2u * t0 * kOnes;
}

// d_j + 16 for the heights just west of word w, from the word's own first column:
//   h(x0-1, j) - h(x0-1, 0) = [sum_{j'=1..j} sigma_y(x0, j')] - [sigma_x(x0, j) - sigma_x(x0, 0)]
__device__ __forceinline__ uint32_t run_start_dq(uint32_t w)
{
    const int x0 = (int)(w & 1u), x1 = (int)((w >> 8) & 1u), x2 = (int)((w >> 16) & 1u), x3 = (int)((w >> 24) & 1u);
    const int y1 = 2 * (int)((w >> 9) & 1u) - 1, y2 = y1 + 2 * (int)((w >> 17) & 1u) - 1, y3 = y2 + 2 * (int)((w >> 25) & 1u) - 1;
    const int d1 = y1 - 2 * (x1 - x0), d2 = y2 - 2 * (x2 - x0), d3 = y3 - 2 * (x3 - x0);
    return 16u | ((uint32_t)(16 + d1) << 8) | ((uint32_t)(16 + d2) << 16) | ((uint32_t)(16 + d3) << 24);
}

__device__ __forceinline__ int warp_inclusive_scan_i32(int v, int lane)
{
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const int u = __shfl_up_sync(0xFFFFFFFFu, v, off);
        if (lane >= off) v += u;
    }
    return v;
}

template <int RUN>
__device__ __forceinline__ void load_run(const uint32_t* __restrict__ p, uint32_t (&w)[RUN])
{
#pragma unroll
    for (int q = 0; q < RUN / 4; ++q) {
        const uint4 v = reinterpret_cast<const uint4*>(p)[q];
        w[4 * q + 0] = v.x; w[4 * q + 1] = v.y; w[4 * q + 2] = v.z; w[4 * q + 3] = v.w;
    }
}

constexpr int kRows2Warps = 8;

// what one pass computes (oct_observe): any combination
enum : int { kObsW2 = 1, kObsCh = 2, kObsCs = 4 };

// heights of the four sites of a word, byte-parallel over its four site rows, from the heights just west of it:
// H_i = H_{i-1} + 2 b_i - 1 per byte (bytes stay within [1, 255]: no carry or borrow between byte lanes, so the
// three-input 32-bit add is four byte adds).  2 b_i is the word's bit 2i of every byte moved to bit 1.
__device__ __forceinline__ void walk_word(uint32_t w, uint32_t& west, uint32_t (&H)[4])
{
    constexpr uint32_t kTwos = 0x02020202u;
    H[0] = west + ((w << 1) & kTwos) - kOnes;
    H[1] = H[0] + ((w >> 1) & kTwos) - kOnes;
    H[2] = H[1] + ((w >> 3) & kTwos) - kOnes;
    H[3] = H[2] + ((w >> 5) & kTwos) - kOnes;
    west = H[3];
}

// One pass over the packed lattice (and the snapshot) for any combination of
//   kObsW2: S1 = sum (h - c), S2 = sum (h - c)^2                         (Eq. (3) :61)
//   kObsCh: S_t = S1, S_s = sum (h_s - c_s), S_ts = sum (h - c)(h_s - c_s) (Eq. (6) :92-98)
//   kObsCs: the six slope-bit sums of :85-88
// RUN words per lane per chunk: 16 for L >= 2048 (chunk = 512 words), 4 below (any L >= 16 works: lanes beyond L/16 idle).
// out (int64): [0..3] = {S1, S2, c, net}; [4..8] = {S_t, S_s, S_ts, c_t, c_s}; [9..14] = {xx, yy, x_t, y_t, x_s, y_s}
template <int WHAT, int RUN>
__device__ __forceinline__ void rows3_body(const RowsParams& P)
{
    constexpr bool W2 = (WHAT & kObsW2) != 0, CH = (WHAT & kObsCh) != 0, CS = (WHAT & kObsCs) != 0;
    constexpr bool NEED_B = CH || CS;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t LW = P.L >> 2;
    const uint32_t wy = blockIdx.x * kRows2Warps + warp;     // word-row of this warp
    long long s1 = 0, s2 = 0, ss = 0, sts = 0;
    unsigned int pc[6] = {0, 0, 0, 0, 0, 0};                 // per thread < 2^32 bits: a thread sees L/8 words of 32 bits per row chunk

    if (wy < LW) {
        const uint32_t* rowA = P.latA + (size_t)wy * LW;
        const uint32_t* rowB = NEED_B ? P.latB + (size_t)wy * LW : nullptr;
        // height just west of site 0 of site row 4*wy, relative to h(0,0):  h(-1,y) = h(0,y) - sigma_x(0,y)
        int carryA = 0, carryB = 0;
        if constexpr (W2 || CH) carryA = P.anchorA[4 * wy] - ((rowA[0] & 1u) ? 1 : -1);
        if constexpr (CH) carryB = P.anchorB[4 * wy] - ((rowB[0] & 1u) ? 1 : -1);
        const uint32_t lanes_used = LW / RUN < 32u ? LW / RUN : 32u;
        const bool on = (uint32_t)lane < lanes_used;

        for (uint32_t wx0 = 0; wx0 < LW; wx0 += 32 * RUN) {
            const uint32_t wx = wx0 + lane * RUN;
            uint32_t wa[RUN], wb[RUN];
            if (on) {
                load_run<RUN>(rowA + wx, wa);
                if constexpr (NEED_B) load_run<RUN>(rowB + wx, wb);
            } else {
#pragma unroll
                for (int k = 0; k < RUN; ++k) { wa[k] = 0x05050505u; wb[k] = 0x05050505u; }   // zero net slope
            }
            if constexpr (CS) {
                if (on) {
                    constexpr uint32_t MX = 0x55555555u;
#pragma unroll
                    for (int k = 0; k < RUN; ++k) {
                        const uint32_t ab = wa[k] & wb[k];
                        pc[0] += __popc(ab & MX); pc[1] += __popc(ab);           // [1], [3], [5] hold x + y until the end
                        pc[2] += __popc(wa[k] & MX); pc[3] += __popc(wa[k]);
                        pc[4] += __popc(wb[k] & MX); pc[5] += __popc(wb[k]);
                    }
                }
            }
            if constexpr (W2 || CH) {
                // heights relative to the (still unknown) height s at the start of this lane's run, kept ENTIRELY in bytes:
                // over a run of <= 64 sites they stay within +-73 of s, so H = e - s + 128 is an unsigned byte and the
                // run's sums are plain DP4A accumulations; the bias comes off once per run
                uint32_t ba = run_start_dq(wa[0]) + 112u * kOnes, bb = 0;      // bytes left_j - s + 128
                if constexpr (CH) bb = run_start_dq(wb[0]) + 112u * kOnes;
                // neighbouring columns differ by one, so H_0^2 + H_1^2 = 2 H_0 H_1 + 1 in every byte: two dot products per word
                // give sum H^2.  (The same trick for sum H -- columns 1 and 3 plus a population count -- and the shifts as
                // high halves of products were measured and are slower: the ALU pipe is the one that is full, profiles/r2_observables.md)
                unsigned int a1 = 0, b1 = 0, qa = 0, qab = 0;                  // sum H_A, sum H_B, sum H_A0 H_A1 + H_A2 H_A3, sum H_A H_B
#pragma unroll
                for (int k = 0; k < RUN; ++k) {
                    uint32_t HA[4], HB[4];
                    walk_word(wa[k], ba, HA);
#pragma unroll
                    for (int i = 0; i < 4; ++i) a1 = __dp4a(HA[i], kOnes, a1);
                    if constexpr (W2) { qa = __dp4a(HA[0], HA[1], qa); qa = __dp4a(HA[2], HA[3], qa); }
                    if constexpr (CH) {
                        walk_word(wb[k], bb, HB);
#pragma unroll
                        for (int i = 0; i < 4; ++i) b1 = __dp4a(HB[i], kOnes, b1);
#pragma unroll
                        for (int i = 0; i < 4; ++i) qab = __dp4a(HA[i], HB[i], qab);
                    }
                }
                constexpr int nn = 16 * RUN;
                constexpr long long n = 16 * RUN;
                const int ra1 = (int)a1 - 128 * nn;                                   // sum (e_A - s_A)
                const int rb1 = (int)b1 - 128 * nn;
                const int totA = (int)(ba & 0xFFu) - 128, totB = (int)(bb & 0xFFu) - 128;   // net slope of site row 0 over the run
                // place the runs: exclusive scan of the runs' net slope of site row 0 (both lattices in one scan: |tot| <= 64 per
                // lane, so the two running sums share a register as 16-bit halves)
                const int incl = warp_inclusive_scan_i32(CH ? totA + totB * 65536 : totA, lane);
                const int last = __shfl_sync(0xFFFFFFFFu, incl, 31);
                const int inclA = CH ? (int)(short)(incl & 0xFFFF) : incl, lastA = CH ? (int)(short)(last & 0xFFFF) : last;
                const int sA = carryA + inclA - totA;               // height at the start of this lane's run (32-bit: heights are int32)
                carryA += lastA;
                if (on) s1 += (long long)sA * (int)n + ra1;
                if constexpr (W2) {
                    const int q = (int)(2u * qa + 8u * RUN - 256u * a1) + 16384 * nn; // sum H^2 = 2 sum (H_0 H_1 + H_2 H_3) + 8 per word; minus the bias: sum (H - 128)^2
                    if (on) s2 += ((long long)sA * sA) * n + (long long)sA * (2 * ra1) + q;
                }
                if constexpr (CH) {
                    const int q = (int)(qab - 128u * (a1 + b1)) + 16384 * nn;         // sum (H_A - 128)(H_B - 128)
                    const int inclB = (incl - inclA) >> 16, lastB = (last - lastA) >> 16;
                    const int sB = carryB + inclB - totB;
                    carryB += lastB;
                    if (on) {
                        ss += (long long)sB * (int)n + rb1;
                        sts += ((long long)sA * sB) * n + (long long)sA * rb1 + (long long)sB * ra1 + q;
                    }
                }
            }
        }
    }

    __shared__ long long red[4][kRows2Warps];
    __shared__ unsigned long long redc[6][kRows2Warps];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        s1 += __shfl_xor_sync(0xFFFFFFFFu, s1, off);
        if constexpr (W2) s2 += __shfl_xor_sync(0xFFFFFFFFu, s2, off);
        if constexpr (CH) { ss += __shfl_xor_sync(0xFFFFFFFFu, ss, off); sts += __shfl_xor_sync(0xFFFFFFFFu, sts, off); }
    }
    if constexpr (CS) {
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const unsigned long long v = __reduce_add_sync(0xFFFFFFFFu, pc[k]);   // a warp's total per row stays far below 2^32
            if (lane == 0) redc[k][warp] = v;
        }
    }
    if (lane == 0) { red[0][warp] = s1; red[1][warp] = s2; red[2][warp] = ss; red[3][warp] = sts; }
    __syncthreads();
    if (threadIdx.x == 0) {
        long long t1 = 0, t2 = 0, t3 = 0, t4 = 0;
        for (int w = 0; w < kRows2Warps; ++w) { t1 += red[0][w]; t2 += red[1][w]; t3 += red[2][w]; t4 += red[3][w]; }
        if constexpr (W2) {
            atomicAdd(&P.out[0], (unsigned long long)t1);
            atomicAdd(&P.out[1], (unsigned long long)t2);
        }
        if constexpr (CH) {
            atomicAdd(&P.out_ch[0], (unsigned long long)t1);
            atomicAdd(&P.out_ch[1], (unsigned long long)t3);
            atomicAdd(&P.out_ch[2], (unsigned long long)t4);
        }
        if (blockIdx.x == 0) {
            if constexpr (W2) { P.out[2] = P.countersA[1]; P.out[3] = P.countersA[0]; }                         // c = h(0,0), net
            if constexpr (CH) { P.out_ch[3] = P.countersA[1]; P.out_ch[4] = (unsigned long long)P.snapB[0]; }         // c_t, c_s
        }
    }
    if constexpr (CS) {
        if (threadIdx.x < 6) {
            unsigned long long t = 0;
            for (int w = 0; w < kRows2Warps; ++w) t += redc[threadIdx.x][w];
            // [1], [3], [5] were counted over both slope bits: take the x part off
            unsigned long long tx = 0;
            if (threadIdx.x & 1) { for (int w = 0; w < kRows2Warps; ++w) tx += redc[threadIdx.x - 1][w]; }
            const int slot = 9 + (int)threadIdx.x;
            atomicAdd(&P.out[slot], t - tx);
        }
    }
}

template <int WHAT, int RUN>
__global__ void __launch_bounds__(kRows2Warps * 32) rows3_kernel(const RowsParams P) { rows3_body<WHAT, RUN>(P); }

// an ensemble: blockIdx.y picks the member (oct_observe_batch)
template <int WHAT, int RUN>
__global__ void __launch_bounds__(kRows2Warps * 32) rows3_batch_kernel(const __grid_constant__ ObsBatchParams BP)
{
    const ObsMember& mb = BP.m[blockIdx.y];
    RowsParams P;
    P.latA = mb.latA; P.latB = mb.latB; P.anchorA = mb.anchorA; P.anchorB = mb.anchorB; P.countersA = mb.countersA;
    P.snapB = mb.snapB; P.heights = nullptr; P.out = mb.out; P.out_ch = mb.out + 4; P.L = BP.L;
    rows3_body<WHAT, RUN>(P);
}

// Heights (a8): the output (16 bytes per site row per word) dwarfs the input, so the lanes take
// *adjacent* words -- every store instruction of the warp writes 512 contiguous bytes -- and the warp
// pays one 32-bit shuffle scan per 32 words (site row 0 only; the other three rows hang off it through
// dq).  UNR independent word-groups are loaded up front for memory-level parallelism.
template <int UNR>
__global__ void __launch_bounds__(kRows2Warps * 32) heights_kernel(const RowsParams P)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t LW = P.L >> 2;
    const uint32_t wy = blockIdx.x * kRows2Warps + warp;
    if (wy >= LW) return;
    const uint32_t* row = P.latA + (size_t)wy * LW;
    const int h00 = (int)(long long)P.countersA[1];
    int carry = P.anchorA[4 * wy] - ((row[0] & 1u) ? 1 : -1) + h00;     // h(-1, 4 wy)
    int* out = P.heights + (size_t)(4 * wy) * P.L;

    for (uint32_t wx0 = 0; wx0 < LW; wx0 += 32 * UNR) {
        uint32_t w[UNR];
#pragma unroll
        for (int k = 0; k < UNR; ++k) {
            const uint32_t wx = wx0 + 32 * k + lane;
            w[k] = wx < LW ? row[wx] : 0x05050505u;                     // zero net slope past a short row
        }
#pragma unroll
        for (int k = 0; k < UNR; ++k) {
            const uint32_t wx = wx0 + 32 * k + lane;
            const int tot = 2 * __popc(w[k] & 0x55u) - 4;
            const int incl = warp_inclusive_scan_i32(tot, lane);
            RowRun st{carry + incl - tot - 16, run_start_dq(w[k])};
            carry += __shfl_sync(0xFFFFFFFFu, incl, 31);
            uint32_t H[4]; int r0;
            word_heights(w[k], st, H, r0);
            if (wx < LW) {
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int4 v = make_int4(r0 + (int)((H[0] >> (8 * j)) & 0xFFu), r0 + (int)((H[1] >> (8 * j)) & 0xFFu),
                                             r0 + (int)((H[2] >> (8 * j)) & 0xFFu), r0 + (int)((H[3] >> (8 * j)) & 0xFFu));
                    __stcs(reinterpret_cast<int4*>(out + (size_t)j * P.L + 4 * wx), v);   // streaming: never re-read here
                }
            }
        }
    }
}

}  // namespace octb

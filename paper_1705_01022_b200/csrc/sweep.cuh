// Sweep kernel, bit-packed window: one launch = one domain-set sweep of a DD scheme of arXiv 1705.01022
// (Sec. 3).  This is the general kernel (every device layer incl. the dead-border schemes, every shape, D up to 256);
// sweep_links.cuh holds the faster link-entry kernel, which serves every device layer for the shapes it is built for
// (D <= 256) and is what AUTO picks there; this one remains the fallback and the second implementation of every parity case.
//
// B200 mapping (differs from the paper's Kepler kernel):
//   * a device-layer domain (D x D sites) is owned by a small *worker group* of WPD
//     warps -- one single warp where the domain has <= 128 thread cells -- instead of one
//     1024-thread block.  The block-layer thread cells (:168) are logical: each lane carries CPT cells
//     per collective step (instruction-level parallelism), and the per-step synchronisation is
//     __syncwarp (WPD = 1), a named barrier over the group, or the CTA barrier when the group is the CTA.
//   * the domain window ((D/4+1)^2 words: D x D sites plus the +x / +y halo, :140, :164) is staged
//     into shared memory in the lattice's own word alignment, odd pitch (:123 "padding by one word").
//   * all random numbers are Philox4x32-10 words generated in registers (one call = 4 steps of one
//     cell); the per-MCS control (origin, permutation, :144/:150) is recomputed by every group from
//     the global stream, so the host does no arithmetic and launches carry only (t, set position).
//   * flips are shared-memory atomic XORs because cells displaced by a random origin share words
//     (:172).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "philox.cuh"

namespace octb {

enum : int { kBlkSync = 0, kBlkDelayed = 1, kBlkDT = 2 };
enum : uint32_t { kDevDTr = 0, kDevDT = 1, kDevDB = 2, kDevCDB = 3, kDevDBh = 4 };

struct SweepParams {
    uint32_t* lat;                  // packed lattice, (L/4)^2 words
    unsigned long long* counters;   // [0] = net deposits (two's complement int64), [1] = h(0,0)
    uint32_t L;
    uint32_t log2L;
    uint32_t t;                     // absolute MCS index of this sweep
    uint32_t si;                    // position of this launch in the set permutation (0..3); dead-border layers: interval index
    uint32_t P16, Q16;              // acceptance thresholds, accept iff r16 < P16 (R18)
    uint32_t dev;                   // device-layer scheme
    uint32_t ndom;                  // domains in this launch
    uint32_t dtr_mask;              // block-layer DT: 0; block-layer DTr (:234, R26): ~0 (the origin also moves)
    uint32_t dead_w;                // dead-border layers: border width in sites (DB 5, cDB 1, or the explicit one; :166, :202, R22/R28)
    uint32_t ka;                    // dead-border layers: t_async = 2^-ka MCS, 2^ka launches (intervals) per sweep (:204-206, R27)
    PhiloxRoundKeys rk;
};

// Bits of packed window word (iw, jw) that belong to sites of the tile [offx, offx + D) x [offy, offy + D) (window
// coordinates).  Dead-border tiles with a border narrower than 4 sites and a free origin share words with their
// neighbours whose other bits the neighbour changes in the same launch (:166 -- the reason for the paper's width 5),
// so such words are written back bit-wise (two atomics) instead of whole.
__device__ __forceinline__ uint32_t tile_bits(uint32_t iw, uint32_t jw, uint32_t offx, uint32_t offy, uint32_t D)
{
    uint32_t m = 0u;
#pragma unroll
    for (uint32_t i = 0; i < 4; ++i) {
        const uint32_t x = 4u * iw + i;
        if (x >= offx && x < offx + D) m |= 0x03030303u << (2u * i);
    }
#pragma unroll
    for (uint32_t j = 0; j < 4; ++j) {
        const uint32_t y = 4u * jw + j;
        if (!(y >= offy && y < offy + D)) m &= ~(0xFFu << (8u * j));
    }
    return m;
}

// write back one window word of a dead-border tile: whole if it holds only this tile's sites (or the border is wide
// enough that foreign bits cannot change, dead_w >= 4), else only this tile's bits.  The neighbouring tile stages the
// same word in with a plain load while this one may be writing it: harmless, because a tile consumes only ITS OWN bits
// of a shared word (the foreign bits belong to dead sites: never tested, never written back), and those bits are
// written by nobody else during the launch.
__device__ __forceinline__ void store_tile_word(uint32_t* ptr, uint32_t word, uint32_t iw, uint32_t jw, uint32_t offx, uint32_t offy,
                                                uint32_t D, uint32_t dead_w)
{
    const uint32_t m = dead_w >= 4u ? 0xFFFFFFFFu : tile_bits(iw, jw, offx, offy, D);
    if (m == 0xFFFFFFFFu) { *ptr = word; return; }
    atomicAnd(ptr, word | ~m);
    atomicOr(ptr, word & m);
}

// Several lattices of one size in one launch (oct_sweep_batch; the paper's curves are ensemble means over n = 20 ... 4367
// independent runs): blockIdx.y picks the member, which brings its own lattice, counters,
// seed and clock.  Everything else (size, scheme, rates) is common and sits in `common`.
constexpr int kMaxBatch = 256;
struct BatchMember {
    uint32_t* lat;
    unsigned long long* counters;
    uint32_t seed_lo, seed_hi;
    uint32_t t;
    uint32_t pad;
};
struct SweepBatchParams {
    SweepParams common;             // lat, counters, t and rk are ignored
    BatchMember m[kMaxBatch];
};

template <int LOG2D, int TCX, int TCY, int WPD_>
struct SweepShape {
    static constexpr int D = 1 << LOG2D;
    static constexpr int CX = 4 << TCX, CY = 4 << TCY;
    static constexpr int NCX = D / CX, NCY = D / CY, NCELL = NCX * NCY;
    static constexpr int NSTEP = CX * CY;                      // collective steps per domain sweep (R12)
    static constexpr int WPD = WPD_;
    static constexpr int G = 32 * WPD;                         // threads per worker group
    static constexpr int CPT = (NCELL + G - 1) / G;            // cells per thread per step
    static constexpr bool PARTIAL = (NCELL % G) != 0;
    static constexpr int DPB = WPD >= 4 ? 1 : 4 / WPD;         // domains per CTA
    static constexpr int NTHREADS = G * DPB;
    static constexpr int NW = D / 4 + 1;                       // window edge in words (halo included)
    static constexpr int PITCH = NW;                           // odd -> rows start in rotating banks
    static constexpr int WORDS = ((NW * PITCH + 3) / 4) * 4;
    static constexpr int SMEM_PER_DOMAIN = (WORDS + NSTEP) * 4;
    static constexpr int SMEM_BYTES = SMEM_PER_DOMAIN * DPB;
    static_assert(CX <= D && CY <= D, "cell larger than domain");
    static_assert(NW * PITCH < 65536, "window index must fit 16 bits");
};

template <int WPD, int DPB>
__device__ __forceinline__ void group_sync(int grp)
{
    if constexpr (WPD == 1) {
        __syncwarp();
    } else if constexpr (DPB == 1) {
        __syncthreads();
    } else {
        asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "n"(32 * WPD) : "memory");
    }
}

// idx-th permutation of (0,1,2,3) in lexicographic order, element `pos` (:144 "a permutation
// shuffled uniformly at each MCS")
__device__ __forceinline__ uint32_t lex_perm4_at(uint32_t idx, uint32_t pos)
{
    uint32_t pool = 0x3210u;   // nibble list of the unused elements, ascending
    uint32_t f = 6, n = 4, e = 0;
#pragma unroll
    for (uint32_t i = 0; i < 4; ++i) {
        const uint32_t j = idx / f;
        idx -= j * f;
        e = (pool >> (4 * j)) & 15u;
        const uint32_t lowmask = (1u << (4 * j)) - 1u;
        pool = (pool & lowmask) | ((pool >> 4) & ~lowmask);
        if (i == pos) break;
        --n;
        if (n > 1) f /= n;
    }
    return e;
}

// Everything a cell needs to carry from the decision to the application of one attempt.
struct Attempt {
    uint32_t loc;    // window word index | bit shift << 16 | (site is the lattice origin) << 24
    int dec;         // +1 deposit, -1 remove, 0 nothing
};

template <class SH>
__device__ __forceinline__ int decide_at(const uint32_t* __restrict__ S, uint32_t sx, uint32_t sy, uint32_t r16,
                                         uint32_t P16, uint32_t Q16, uint32_t& loc)
{
    const uint32_t i = sx & 3u, j = sy & 3u;
    const uint32_t widx = (sy >> 2) * SH::PITCH + (sx >> 2);
    const uint32_t sh = 2u * (4u * j + i);
    const uint32_t A = S[widx];
    const uint32_t own = (A >> sh) & 3u;                    // bit0 sigma_x(x,y), bit1 sigma_y(x,y)
    uint32_t east, north;                                   // sigma_x(x+1,y), sigma_y(x,y+1)
    if (i == 3u) east = (S[widx + 1] >> (8u * j)) & 1u;
    else         east = (A >> (sh + 2u)) & 1u;
    if (j == 3u) north = (S[widx + SH::PITCH] >> (2u * i + 1u)) & 1u;
    else         north = (A >> (sh + 9u)) & 1u;
    loc = widx | (sh << 16);
    // Eq. (1) :27-34: local minimum (sx, sx_east, sy, sy_north) = (0,1,0,1), maximum (1,0,1,0)
    const bool is_min = (own == 0u) & (east == 1u) & (north == 1u);
    const bool is_max = (own == 3u) & (east == 0u) & (north == 0u);
    return (is_min && r16 < P16) ? 1 : ((is_max && r16 < Q16) ? -1 : 0);
}

template <class SH>
__device__ __forceinline__ void apply_at(uint32_t* S, uint32_t loc)
{
    const uint32_t widx = loc & 0xFFFFu, sh = (loc >> 16) & 31u;
    const uint32_t i = (sh >> 1) & 3u, j = sh >> 3;
    uint32_t mA = 3u << sh;
    if (i != 3u) mA |= 4u << sh;
    if (j != 3u) mA |= 0x200u << sh;
    atomicXor(&S[widx], mA);
    if (i == 3u) atomicXor(&S[widx + 1], 1u << (8u * j));
    if (j == 3u) atomicXor(&S[widx + SH::PITCH], 2u << (2u * i));
}

template <int LOG2D, int TCX, int TCY, int BLK, int WPD>
__global__ void __launch_bounds__(SweepShape<LOG2D, TCX, TCY, WPD>::NTHREADS)
sweep_kernel(const __grid_constant__ SweepParams P)
{
    using SH = SweepShape<LOG2D, TCX, TCY, WPD>;
    constexpr int D = SH::D, CX = SH::CX, CY = SH::CY, G = SH::G, CPT = SH::CPT, NW = SH::NW, PITCH = SH::PITCH;
    constexpr uint32_t LOG2NCX = LOG2D - TCX - 2;

    extern __shared__ uint32_t smem_raw[];
    const int grp = threadIdx.x / G;                 // worker group inside the CTA
    const uint32_t tg = threadIdx.x % G;             // thread inside the group
    uint32_t* S = smem_raw + grp * (SH::SMEM_PER_DOMAIN / 4);
    uint32_t* BT = S + SH::WORDS;                    // block-step words of this domain sweep

    const uint32_t L = P.L, Lm = L - 1u, t = P.t;
    const uint32_t dom = blockIdx.x * SH::DPB + grp;
    if (dom >= P.ndom) return;                       // whole group leaves together (own barrier id)

    // ---- a1: per-MCS control from the global stream (:144, :150; R10) --------------------------
    // dead-border layers with t_async = 2^-ka MCS (:204-206, R27): the launch is interval P.si of the sweep, with its
    // own origin (global stream c0 = interval), 1/2^ka of the collective steps, streams keyed by set = interval
    const bool dead = P.dev > kDevDT;
    uint32_t Gw[4];
    philox4x32_10(dead ? P.si : 0u, 0u, kTagGlobal << 30, t, P.rk, Gw);
    uint32_t gx, gy, set, dead_w;
    if (P.dev <= kDevDT) {
        const uint32_t Ox = P.dev == kDevDTr ? (Gw[0] & Lm) : 0u, Oy = P.dev == kDevDTr ? (Gw[1] & Lm) : 0u;
        set = lex_perm4_at(Gw[2] % 24u, P.si);
        const uint32_t lnt = P.log2L - LOG2D - 1u;                      // log2 tiles per edge
        const uint32_t I = dom & ((1u << lnt) - 1u), J = dom >> lnt;
        gx = (Ox + (I << (LOG2D + 1)) + ((set & 1u) << LOG2D)) & Lm;
        gy = (Oy + (J << (LOG2D + 1)) + ((set >> 1) << LOG2D)) & Lm;
        dead_w = 0u;
    } else {
        uint32_t Ox = Gw[0] & Lm, Oy = Gw[1] & Lm;
        if (P.dev == kDevCDB) { Ox &= ~3u; Oy &= ~3u; }                 // :166 coarse grid
        set = P.si;                                                     // interval index keys the streams (R27)
        const uint32_t lnt = P.log2L - LOG2D;
        const uint32_t I = dom & ((1u << lnt) - 1u), J = dom >> lnt;
        gx = (Ox + (I << LOG2D)) & Lm;
        gy = (Oy + (J << LOG2D)) & Lm;
        dead_w = P.dead_w;                                              // :166, R22/R28
    }
    const uint32_t offx = gx & 3u, offy = gy & 3u;
    const uint32_t LW = L >> 2, LWm = LW - 1u, wx0 = gx >> 2, wy0 = gy >> 2;
    // is the lattice origin (0,0) inside this domain?  (anchor tracking, R20)
    const uint32_t x00 = (0u - gx) & Lm, y00 = (0u - gy) & Lm;
    const bool has00 = x00 < (uint32_t)D && y00 < (uint32_t)D;

    // ---- a2: stage-in (:164) ---------------------------------------------------------------------
    // Dead-border layers: window words past the last column / row that holds one of this tile's active sites (or their
    // E / N links) belong to the next tile, which writes them in this same launch.  They are neither tested nor written
    // back here, so they are not loaded either (zeros stand in), as kept() does in sweep_links.cuh: no cross-CTA
    // read of a word another CTA is writing.
    const uint32_t ncol = dead ? ((offx + (uint32_t)D - dead_w) >> 2) + 1u : (uint32_t)NW;
    const uint32_t nrow = dead ? ((offy + (uint32_t)D - dead_w) >> 2) + 1u : (uint32_t)NW;
    for (uint32_t idx = tg; idx < (uint32_t)(NW * NW); idx += G) {
        const uint32_t j = idx / NW, i = idx - j * NW;
        S[j * PITCH + i] = (i < ncol && j < nrow) ? P.lat[(size_t)((wy0 + j) & LWm) * LW + ((wx0 + i) & LWm)] : 0u;
    }
    // ---- a3: block-step table (:170, :172; R13/R17/R24) ------------------------------------------
    const uint32_t c2b = (kTagBlock << 30) | (set << 28) | dom, c2c = (kTagCell << 30) | (set << 28) | dom;
    for (uint32_t q = tg; q < (uint32_t)(SH::NSTEP / 4); q += G) {
        uint32_t o[4];
        philox4x32_10(q, 0u, c2b, t, P.rk, o);
        BT[4 * q + 0] = o[0]; BT[4 * q + 1] = o[1]; BT[4 * q + 2] = o[2]; BT[4 * q + 3] = o[3];
    }
    group_sync<WPD, SH::DPB>(grp);

    // ---- a4-a6: collective single-hit steps (:168) -----------------------------------------------
    const uint32_t P16 = P.P16, Q16 = P.Q16;
    int net = 0, d00 = 0;
    const uint32_t dead_lim = (uint32_t)D - dead_w;

    const uint32_t k4_per = dead ? (uint32_t)(SH::NSTEP / 4) >> P.ka : (uint32_t)(SH::NSTEP / 4);   // steps of this interval
    const uint32_t k4_begin = dead ? P.si * k4_per : 0u, k4_end = k4_begin + k4_per;
#pragma unroll 1
    for (uint32_t k4 = k4_begin; k4 < k4_end; ++k4) {
        uint32_t rw[CPT][4];
#pragma unroll
        for (int j = 0; j < CPT; ++j) philox4x32_10(k4, tg + j * G, c2c, t, P.rk, rw[j]);

#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
            const uint32_t Bw = BT[4 * k4 + kk];
            Attempt at[CPT];
            if constexpr (BLK == kBlkDT) {
                // :170 one random quadrant for all cells of the block in this step (R17)
                // block-layer DTr (:234, R26) adds the per-step origin of block-layer DB, cells wrap (R14)
                const uint32_t qx = ((Bw >> 16) & 1u) * (CX / 2) + (Bw & (CX - 1) & P.dtr_mask);
                const uint32_t qy = ((Bw >> 17) & 1u) * (CY / 2) + ((Bw >> 8) & (CY - 1) & P.dtr_mask);
#pragma unroll
                for (int j = 0; j < CPT; ++j) {
                    const uint32_t c = tg + j * G, w = rw[j][kk];
                    const uint32_t x = ((c & (SH::NCX - 1)) * CX + qx + (w & (CX / 2 - 1))) & (D - 1);
                    const uint32_t y = ((c >> LOG2NCX) * CY + qy + ((w >> 8) & (CY / 2 - 1))) & (D - 1);
                    int dec = 0; uint32_t loc = 0;
                    const bool live = (!SH::PARTIAL || c < (uint32_t)SH::NCELL) && x < dead_lim && y < dead_lim;
                    if (live) dec = decide_at<SH>(S, x + offx, y + offy, w >> 16, P16, Q16, loc);
                    if (dec) {
                        apply_at<SH>(S, loc);
                        net += dec;
                        if (has00 && x == x00 && y == y00) d00 += 2 * dec;
                    }
                }
                group_sync<WPD, SH::DPB>(grp);
            } else {
                // :172 DB with a random cell origin per step; cells wrap inside the domain (R14)
                const uint32_t ox = Bw & (CX - 1), oy = (Bw >> 8) & (CY - 1);
                uint32_t cls[CPT];
#pragma unroll
                for (int j = 0; j < CPT; ++j) {
                    const uint32_t c = tg + j * G, w = rw[j][kk];
                    const uint32_t lx = w & (CX - 1), ly = (w >> 8) & (CY - 1);
                    const uint32_t x = ((c & (SH::NCX - 1)) * CX + lx + ox) & (D - 1);
                    const uint32_t y = ((c >> LOG2NCX) * CY + ly + oy) & (D - 1);
                    const bool live = (!SH::PARTIAL || c < (uint32_t)SH::NCELL) && x < dead_lim && y < dead_lim;
                    const uint32_t is00 = (has00 && x == x00 && y == y00) ? 1u : 0u;
                    if constexpr (BLK == kBlkSync) {
                        // "ignoring borders" (:174) made order-free: decide on the step's initial state (R16)
                        at[j].dec = 0; at[j].loc = 0;
                        if (live) at[j].dec = decide_at<SH>(S, x + offx, y + offy, w >> 16, P16, Q16, at[j].loc);
                        at[j].loc |= is00 << 24;
                    } else {
                        cls[j] = live ? (uint32_t)(lx == CX - 1) + (uint32_t)(ly == CY - 1) : 3u;
                        at[j].loc = (x + offx) | ((y + offy) << 12) | (is00 << 24);
                    }
                }
                if constexpr (BLK == kBlkSync) {
                    group_sync<WPD, SH::DPB>(grp);
#pragma unroll
                    for (int j = 0; j < CPT; ++j)
                        if (at[j].dec) {
                            apply_at<SH>(S, at[j].loc);
                            net += at[j].dec;
                            if (at[j].loc >> 24) d00 += 2 * at[j].dec;
                        }
                    group_sync<WPD, SH::DPB>(grp);
                } else {
                    // delayed borders (:174): bulk, then edges, then corners
#pragma unroll
                    for (uint32_t phase = 0; phase < 3; ++phase) {
#pragma unroll
                        for (int j = 0; j < CPT; ++j)
                            if (cls[j] == phase) {
                                uint32_t loc;
                                const int dec = decide_at<SH>(S, at[j].loc & 0xFFFu, (at[j].loc >> 12) & 0xFFFu,
                                                              rw[j][kk] >> 16, P16, Q16, loc);
                                if (dec) {
                                    apply_at<SH>(S, loc);
                                    net += dec;
                                    if (at[j].loc >> 24) d00 += 2 * dec;
                                }
                            }
                        group_sync<WPD, SH::DPB>(grp);
                    }
                }
            }
        }
    }

    // ---- a7: stage-out (:164).  Whole words; for dead-border schemes the words that also hold the
    // next tile's sites are never modified here and are not written (:166) ------------------------
    for (uint32_t idx = tg; idx < (uint32_t)(NW * NW); idx += G) {
        const uint32_t j = idx / NW, i = idx - j * NW;
        if (i < ncol && j < nrow) {
            uint32_t* ptr = P.lat + (size_t)((wy0 + j) & LWm) * LW + ((wx0 + i) & LWm);
            if (dead) store_tile_word(ptr, S[j * PITCH + i], i, j, offx, offy, (uint32_t)D, dead_w);
            else *ptr = S[j * PITCH + i];
        }
    }

    // counters: net deposits (one atomic per warp) and the tracked height of site (0,0)
    net = __reduce_add_sync(0xFFFFFFFFu, net);
    if ((threadIdx.x & 31) == 0 && net != 0) atomicAdd(&P.counters[0], (unsigned long long)(long long)net);
    if (d00 != 0) atomicAdd(&P.counters[1], (unsigned long long)(long long)d00);
}

}  // namespace octb

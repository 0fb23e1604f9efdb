// Sweep kernel, link-entry layout: one launch = one domain-set sweep of any device-layer scheme of
// arXiv 1705.01022 (DTr / DT: Sec. 3.0.2-3.0.3; DB / cDB / DBh: Sec. 3.0.1, :133-140, :166)
// with any of the single-hit block layers (Sec. 3.1, :168-174), for device-layer domains of D <= 128 sites.
//
// Why a second layout (profiles/r1_a_*.md): on the bit-packed window the update test costs ~115 SASS
// instructions per attempt, almost all of them shift/mask arithmetic and shared-memory atomics, and the
// ALU pipe binds.  Here the window is unpacked ONCE per domain sweep into one 32-bit *entry* per site that
// carries the four links of that site, one byte each:
//      byte 0  W = sigma_x(x,y)     byte 1  E = sigma_x(x+1,y)
//      byte 2  S = sigma_y(x,y)     byte 3  N = sigma_y(x,y+1)                      (:140, R3)
// so that
//   * the eligibility test of Eq. (1) (:27-34) is one LDS.32 and one compare: local minimum
//     (W,E,S,N) = (0,1,0,1) <=> entry == 0x01000100, local maximum <=> entry == 0x00010001;
//   * an accepted update is five plain stores: the site's own entry and one byte in each of the four
//     neighbouring entries (every link is stored twice, once per end site).  No atomics are needed:
//     a link can only be changed by an update at one of its two end sites, two nearest-neighbour sites
//     are never updated in the same phase (:174, R15/R16), and byte stores leave the other bytes of a
//     word alone.  Entries of sites outside the active D x D square (halo and alignment padding) take
//     stray byte writes in their E/N bytes only, which are never read and never written back.
//   * the window is kept in the lattice's own 4-site word alignment (pitch D+4 entries), so stage-in
//     expands a packed word into four 128-bit stores and stage-out gathers it back from four 128-bit
//     loads with multiply-shift bit gathers.
// Everything else (Philox streams, per-MCS control, cell geometry, phases) is as in sweep.cuh and
// follows the same readings R10-R19 of DESIGN.md.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "philox.cuh"
#include "sweep.cuh"

namespace octb {

constexpr uint32_t kEntryMin = 0x01000100u;   // (W,E,S,N) = (0,1,0,1): local minimum, Eq. (1)
constexpr uint32_t kEntryMax = 0x00010001u;   // (1,0,1,0): local maximum

template <int LOG2D, int TCX, int TCY, int WPD_, int DPB_>
struct LinkShape {
    static constexpr int D = 1 << LOG2D;
    static constexpr int CX = 4 << TCX, CY = 4 << TCY;
    static constexpr int NCX = D / CX, NCY = D / CY, NCELL = NCX * NCY;
    static constexpr int NSTEP = CX * CY;                 // collective steps per domain sweep (R12)
    static constexpr int WPD = WPD_, DPB = DPB_;
    static constexpr int G = 32 * WPD;                    // threads per worker group (one domain)
    static constexpr int CPT = NCELL / G;                 // cells per thread per collective step
    static constexpr int NTHREADS = G * DPB;
    static constexpr int NW = D / 4 + 1;                  // window edge in packed words (halo included)
    static constexpr int P = 4 * NW;                      // entries per row (multiple of 4: 128-bit rows)
    static constexpr int ROWS = 4 * NW + 1;               // one spare row below row 0 for stray S-writes
    static constexpr int ENTRY_WORDS = ROWS * P;
    static constexpr int SMEM_PER_DOMAIN = (ENTRY_WORDS + NSTEP) * 4;
    static constexpr int SMEM_BYTES = SMEM_PER_DOMAIN * DPB;
    static_assert(LOG2D <= 7, "x and y are decoded in 8-bit fields: D + CX - 2 must stay below 256");
    static_assert(NCELL % G == 0 && CPT >= 1, "every thread carries the same number of cells");
    static_assert(CX <= D && CY <= D, "cell larger than domain");
};

// bits 0,2,4,6 of b -> bit 0 of bytes 0,1,2,3 (multiply-shift scatter; partial products never collide
// in a way that carries into a kept bit)
__device__ __forceinline__ uint32_t scatter4(uint32_t b) { return ((b & 0x55u) * 0x41041u) & 0x01010101u; }

// Expand packed word A (with its east neighbour Ew and north neighbour Nw) into 16 entries.
template <class SH>
__device__ __forceinline__ void expand_word(uint32_t* __restrict__ S, uint32_t iw, uint32_t jw, uint32_t A,
                                            uint32_t Ew, uint32_t Nw)
{
    uint32_t sy[5];
#pragma unroll
    for (int j = 0; j < 4; ++j) sy[j] = scatter4(A >> (8 * j + 1));
    sy[4] = scatter4(Nw >> 1);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint32_t sx = scatter4(A >> (8 * j));
        const uint32_t sxe = (sx >> 8) | (((Ew >> (8 * j)) & 1u) << 24);   // sigma_x of the site to the east
        const uint32_t t0 = __byte_perm(sx, sxe, 0x5140), t1 = __byte_perm(sx, sxe, 0x7362);
        const uint32_t u0 = __byte_perm(sy[j], sy[j + 1], 0x5140), u1 = __byte_perm(sy[j], sy[j + 1], 0x7362);
        uint4 q;
        q.x = __byte_perm(t0, u0, 0x5410); q.y = __byte_perm(t0, u0, 0x7632);
        q.z = __byte_perm(t1, u1, 0x5410); q.w = __byte_perm(t1, u1, 0x7632);
        *reinterpret_cast<uint4*>(S + (4 * jw + j) * SH::P + 4 * iw) = q;
    }
}

// Gather the own links (bytes 0 and 2) of 16 entries back into one packed word.
template <class SH>
__device__ __forceinline__ uint32_t gather_word(const uint32_t* __restrict__ S, uint32_t iw, uint32_t jw)
{
    uint32_t word = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint4 q = *reinterpret_cast<const uint4*>(S + (4 * jw + j) * SH::P + 4 * iw);
        const uint32_t z = q.x + 4u * q.y + 16u * q.z + 64u * q.w;       // W bits at 0,2,4,6; S bits at 16,18,20,22
        const uint32_t rb = (z & 0x55u) | ((z >> 15) & 0xAAu);
        word |= rb << (8 * j);
    }
    return word;
}

// entry index y*P + x of the site packed as v = x | y << 8 (fields may hold x + D, y + D: cells wrap inside
// the domain, R14): mask both fields at once, then y*P + x = vm + y*(P - 256)
template <class SH>
__device__ __forceinline__ uint32_t site_index(uint32_t v)
{
    const uint32_t vm = v & (uint32_t)((SH::D - 1) | ((SH::D - 1) << 8));
    return (vm >> 8) * (uint32_t)(SH::P - 256) + vm;
}

// First moment sum_x x * b(x) of the sigma_x bits of packed window word (iw, .), x = 4*iw + i.  The sweep
// does not count its accepted updates: inside a window row the heights of the sites west and east of the
// active span are fixed during the launch, so sum_x delta b(x) = 0 and the rise of the surface is
// sum_sites delta h = -2 sum x * delta b(x); every deposit raises one site by 2, hence
//     deposits - removals = sum over window words of (moment before - moment after).
__device__ __forceinline__ int x_moment(uint32_t word, uint32_t iw)
{
    const uint32_t m = word & 0x55555555u;
    return (int)(4u * iw * __popc(m) + __popc(m & 0x44444444u) + 2u * __popc(m & 0x50505050u));
}

// Carry out an accepted update at entry index `i` (relative to Sb): the site's four links flip.
// up = true: deposition (minimum -> maximum), false: removal.
template <class SH>
__device__ __forceinline__ void flip_links(uint32_t* Sb, uint32_t i, bool up)
{
    unsigned char* B = reinterpret_cast<unsigned char*>(Sb + i);
    const unsigned char v1 = up ? 1 : 0, v0 = up ? 0 : 1;
    Sb[i] = up ? kEntryMax : kEntryMin;
    B[-4 + 1] = v1;                 // west neighbour's E link  = sigma_x(x,y)
    B[+4 + 0] = v0;                 // east neighbour's W link  = sigma_x(x+1,y)
    B[-4 * SH::P + 3] = v1;         // south neighbour's N link = sigma_y(x,y)
    B[+4 * SH::P + 2] = v0;         // north neighbour's S link = sigma_y(x,y+1)
}

// Acceptance rule of one launch.  ONEDIR: only one of p, q is non-zero (always so for the sync variant),
// so a single entry pattern is tested and the stored values are launch constants; ALWAYS: that live
// threshold is 65536 (p = 1 or q = 1) and the 16-bit comparison is dropped as well.
template <bool ONEDIR, bool ALWAYS>
struct Rule {
    uint32_t P16, Q16, target, T16;
    bool dep;
    __device__ __forceinline__ Rule(uint32_t p16, uint32_t q16)
        : P16(p16), Q16(q16), target(q16 == 0u ? kEntryMin : kEntryMax), T16(q16 == 0u ? p16 : q16), dep(q16 == 0u) {}
    // decision for entry value e and attempt word w: 0 nothing, +1 deposit, -1 remove
    __device__ __forceinline__ int decide(uint32_t e, uint32_t w) const
    {
        if constexpr (ONEDIR) {
            bool acc = e == target;
            if constexpr (!ALWAYS) acc = acc && (w >> 16) < T16;
            return acc ? (dep ? 1 : -1) : 0;
        } else {
            const uint32_t r16 = w >> 16;
            return (e == kEntryMin && r16 < P16) ? 1 : ((e == kEntryMax && r16 < Q16) ? -1 : 0);
        }
    }
    template <class SH>
    __device__ __forceinline__ void apply(uint32_t* Sb, uint32_t i, int d) const
    {
        if constexpr (ONEDIR) { if (d != 0) flip_links<SH>(Sb, i, dep); }
        else { if (d != 0) flip_links<SH>(Sb, i, d > 0); }
    }
};

// The collective single-hit steps of one domain sweep (:168-174).
// DEAD: dead-border device layer (:135): attempts whose domain-local x or y is >= dead_lim are not carried out.
template <class SH, int BLK, bool ONEDIR, bool ALWAYS, bool DEAD>
__device__ __forceinline__ void run_steps(uint32_t* __restrict__ Sb, const uint32_t* __restrict__ BT, uint32_t tg, int grp,
                                         uint32_t c2c, uint32_t t, const PhiloxRoundKeys& rk, uint32_t P16, uint32_t Q16, uint32_t dtr_mask,
                                         uint32_t dead_lim, uint32_t k4_begin, uint32_t k4_end)
{
    constexpr int CX = SH::CX, CY = SH::CY, G = SH::G, CPT = SH::CPT;
    constexpr uint32_t LOG2NCX = 0 + (SH::NCX == 1 ? 0 : SH::NCX == 2 ? 1 : SH::NCX == 4 ? 2 : SH::NCX == 8 ? 3 : SH::NCX == 16 ? 4 : 5);
    static_assert((1 << LOG2NCX) == SH::NCX, "NCX must be a power of two <= 32");
    // x in bits 0-7, y in bits 8-15 of one register: the attempt word, the block-step word and the cell
    // origin all use this packing, so selecting a site is mask + 3-input add (R13/R14/R19)
    constexpr uint32_t FM = BLK == kBlkDT ? (uint32_t)((CX / 2 - 1) | ((CY / 2 - 1) << 8)) : (uint32_t)((CX - 1) | ((CY - 1) << 8));

    uint32_t cellc[CPT];
#pragma unroll
    for (int j = 0; j < CPT; ++j) {
        const uint32_t c = tg + j * G;
        cellc[j] = ((c & (SH::NCX - 1)) * CX) | (((c >> LOG2NCX) * CY) << 8);
    }
    const Rule<ONEDIR, ALWAYS> rule(P16, Q16);

    // decision for the site packed in v (x | y << 8 before wrapping); idx receives its entry index
    auto decide_site = [&](uint32_t v, uint32_t w, uint32_t& idx) -> int {
        idx = site_index<SH>(v);
        if constexpr (DEAD) {
            const uint32_t vm = v & (uint32_t)((SH::D - 1) | ((SH::D - 1) << 8));
            if ((vm & 0xFFu) >= dead_lim || (vm >> 8) >= dead_lim) return 0;      // dead border: not carried out
        }
        return rule.decide(Sb[idx], w);
    };

    // a few groups of four steps per loop trip: the next groups' Philox rounds fill the issue slots the current
    // group's shared-memory round trips leave open (+3 % at D = 64, +8 % at D = 128 over no unrolling)
    constexpr int kUnrollK4 = CPT >= 4 ? 2 : 8 / CPT;
#pragma unroll kUnrollK4
    for (uint32_t k4 = k4_begin; k4 < k4_end; ++k4) {
        uint32_t rw[CPT][4];
#pragma unroll
        for (int j = 0; j < CPT; ++j) philox4x32_10(k4, tg + j * G, c2c, t, rk, rw[j]);

        const uint4 bq = *reinterpret_cast<const uint4*>(BT + 4 * k4);   // one broadcast load for four steps
        const uint32_t bw4[4] = {bq.x, bq.y, bq.z, bq.w};
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
            const uint32_t Bw = bw4[kk];
            uint32_t idx[CPT];
            if constexpr (BLK == kBlkSync) {
                // "ignoring borders" (:174) made order-free (R16): all cells decide on the state at the start
                // of the step, then all accepted updates are carried out
                const uint32_t sc = Bw & FM;
                int dec[CPT];
#pragma unroll
                for (int j = 0; j < CPT; ++j) {
                    const uint32_t w = rw[j][kk];
                    dec[j] = decide_site((w & FM) + cellc[j] + sc, w, idx[j]);
                }
                group_sync<SH::WPD, SH::DPB>(grp);
#pragma unroll
                for (int j = 0; j < CPT; ++j) rule.template apply<SH>(Sb, idx[j], dec[j]);
                group_sync<SH::WPD, SH::DPB>(grp);
            } else if constexpr (BLK == kBlkDelayed) {
                // delayed borders (:174): bulk, then edges, then corners (R15)
                const uint32_t sc = Bw & FM;
                uint32_t cls[CPT], vv[CPT];
#pragma unroll
                for (int j = 0; j < CPT; ++j) {
                    const uint32_t f = rw[j][kk] & FM;
                    vv[j] = f + cellc[j] + sc;
                    cls[j] = (uint32_t)((f & 0xFFu) == (uint32_t)(CX - 1)) + (uint32_t)((f >> 8) == (uint32_t)(CY - 1));
                }
#pragma unroll
                for (uint32_t phase = 0; phase < 3; ++phase) {
                    int dec[CPT];                    // cells of one phase never touch common links (R15): loads first
#pragma unroll
                    for (int j = 0; j < CPT; ++j) dec[j] = cls[j] == phase ? decide_site(vv[j], rw[j][kk], idx[j]) : 0;
#pragma unroll
                    for (int j = 0; j < CPT; ++j) rule.template apply<SH>(Sb, idx[j], dec[j]);
                    group_sync<SH::WPD, SH::DPB>(grp);
                }
            } else {
                // block-layer DT (:170): one random quadrant of every cell per step (R17).  The cells of a step
                // cannot interact, so all loads go first and the stores follow (no load waits behind a store)
                // (block-layer DTr, :234 / R26: plus the per-step origin of block-layer DB; site_index wraps, R14)
                const uint32_t qc = ((((Bw >> 16) & 1u) * (CX / 2)) | ((((Bw >> 17) & 1u) * (CY / 2)) << 8))
                                    + (Bw & dtr_mask & (uint32_t)((CX - 1) | ((CY - 1) << 8)));
                int dec[CPT];
#pragma unroll
                for (int j = 0; j < CPT; ++j) {
                    const uint32_t w = rw[j][kk];
                    dec[j] = decide_site((w & FM) + cellc[j] + qc, w, idx[j]);
                }
#pragma unroll
                for (int j = 0; j < CPT; ++j) rule.template apply<SH>(Sb, idx[j], dec[j]);
                group_sync<SH::WPD, SH::DPB>(grp);
            }
        }
    }
}

// number of set W links of the sites (0..x00, y00) of the domain: h(x00,y00) minus the height of the
// inactive site west of the row start, up to a constant (used before and after the sweep, R20)
template <class SH>
__device__ __forceinline__ int row_links_up(const uint32_t* Sb, uint32_t x00, uint32_t y00, uint32_t tg)
{
    int n = 0;
    for (uint32_t x = tg; x <= x00; x += SH::G) n += (int)(Sb[y00 * SH::P + x] & 1u);
    return n;
}

// DEAD = false: tiled device layers DTr / DT (four launches per MCS, one per domain set);
// DEAD = true : dead-border device layers DB / cDB / DBh (all tiles in one launch; the rim of width dead_w is
//               never updated, and words shared with the next tile are neither counted nor written, :166).
template <int LOG2D, int TCX, int TCY, int BLK, int WPD, int DPB, bool DEAD>
__global__ void __launch_bounds__(LinkShape<LOG2D, TCX, TCY, WPD, DPB>::NTHREADS)
sweep_links_kernel(const __grid_constant__ SweepParams P)
{
    using SH = LinkShape<LOG2D, TCX, TCY, WPD, DPB>;
    constexpr int D = SH::D, G = SH::G, NW = SH::NW;

    extern __shared__ __align__(16) uint32_t smem_raw[];
    const int grp = threadIdx.x / G;                 // worker group inside the CTA
    const uint32_t tg = threadIdx.x % G;             // thread inside the group
    uint32_t* S0 = smem_raw + grp * (SH::SMEM_PER_DOMAIN / 4);
    uint32_t* S = S0 + SH::P;                        // row 0 of the window (one spare row below it)
    uint32_t* BT = S0 + SH::ENTRY_WORDS;             // block-step words of this domain sweep

    const uint32_t L = P.L, Lm = L - 1u, t = P.t;
    const uint32_t dom = blockIdx.x * DPB + grp;
    if (dom >= P.ndom) return;                       // whole group leaves together (own barrier id)

    // ---- a1: per-MCS control from the global stream (:144, :150; R10) --------------------------
    const bool half = DEAD && P.dev == kDevDBh;      // DB with t_async = 1/2: this launch is interval P.si (R27)
    uint32_t Gw[4];
    philox4x32_10(half ? P.si : 0u, 0u, kTagGlobal << 30, t, P.rk, Gw);
    uint32_t gx, gy, set, dead_w;
    if constexpr (!DEAD) {
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
        set = half ? P.si : 0u;
        const uint32_t lnt = P.log2L - LOG2D;
        const uint32_t I = dom & ((1u << lnt) - 1u), J = dom >> lnt;
        gx = (Ox + (I << LOG2D)) & Lm;
        gy = (Oy + (J << LOG2D)) & Lm;
        dead_w = P.dev == kDevCDB ? 1u : 5u;                            // :166, R22
    }
    const uint32_t offx = gx & 3u, offy = gy & 3u;
    const uint32_t LW = L >> 2, LWm = LW - 1u, wx0 = gx >> 2, wy0 = gy >> 2;
    uint32_t* Sb = S + offy * SH::P + offx;          // entry of the domain's site (0,0)
    // window words this domain counts and writes back: all of them, or (dead border) only those that hold no
    // site of the next tile -- the last active site's E / N links still lie inside them (:166)
    const uint32_t ncol = DEAD ? ((offx + (uint32_t)D - dead_w) >> 2) + 1u : (uint32_t)NW;
    const uint32_t nrow = DEAD ? ((offy + (uint32_t)D - dead_w) >> 2) + 1u : (uint32_t)NW;

    // ---- a2: stage-in (:164): packed words -> link entries -------------------------------------
    int net = 0;                                     // deposits - removals, from the x-moments (see x_moment)
    {
        constexpr int NIT = (NW * NW + G - 1) / G;   // words per thread; all loads are issued before the first use
        uint32_t A[NIT], Ew[NIT], Nw[NIT];
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const uint32_t idx = tg + it * G;
            if (idx < (uint32_t)(NW * NW)) {
                const uint32_t jw = idx / NW, iw = idx - jw * NW;
                const size_t r0 = (size_t)((wy0 + jw) & LWm) * LW, r1 = (size_t)((wy0 + jw + 1u) & LWm) * LW;
                const uint32_t c0 = (wx0 + iw) & LWm, c1 = (wx0 + iw + 1u) & LWm;
                A[it] = P.lat[r0 + c0]; Ew[it] = P.lat[r0 + c1]; Nw[it] = P.lat[r1 + c0];
            }
        }
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const uint32_t idx = tg + it * G;
            if (idx < (uint32_t)(NW * NW)) {
                const uint32_t jw = idx / NW, iw = idx - jw * NW;
                expand_word<SH>(S, iw, jw, A[it], Ew[it], Nw[it]);
                if (!DEAD || (iw < ncol && jw < nrow)) net += x_moment(A[it], iw);
            }
        }
    }
    // ---- a3: block-step table (:170, :172; R13/R17/R24) ----------------------------------------
    const uint32_t c2b = (kTagBlock << 30) | (set << 28) | dom, c2c = (kTagCell << 30) | (set << 28) | dom;
    for (uint32_t q = tg; q < (uint32_t)(SH::NSTEP / 4); q += G) {
        uint32_t o[4];
        philox4x32_10(q, 0u, c2b, t, P.rk, o);
        BT[4 * q + 0] = o[0]; BT[4 * q + 1] = o[1]; BT[4 * q + 2] = o[2]; BT[4 * q + 3] = o[3];
    }
    group_sync<WPD, DPB>(grp);

    // is the lattice origin (0,0) an active site of this domain?  (anchor tracking, R20)
    const uint32_t x00 = (0u - gx) & Lm, y00 = (0u - gy) & Lm;
    const bool has00 = x00 < (uint32_t)D && y00 < (uint32_t)D;
    int d00 = 0;
    if (has00) {                                     // group-uniform branch
        d00 = -row_links_up<SH>(Sb, x00, y00, tg);
        group_sync<WPD, DPB>(grp);                   // the first phase may write at once
    }

    // ---- a4-a6: collective single-hit steps (:168) ---------------------------------------------
    // launch-uniform specialisation of the acceptance rule (the sync variant is only used with p*q = 0, R16)
    const bool onedir = BLK == kBlkSync || P.P16 == 0u || P.Q16 == 0u;
    const uint32_t T16 = P.Q16 == 0u ? P.P16 : P.Q16;
    const uint32_t dead_lim = (uint32_t)D - dead_w;
    const uint32_t k4_begin = half ? P.si * (uint32_t)(SH::NSTEP / 8) : 0u;
    const uint32_t k4_end = half ? k4_begin + (uint32_t)(SH::NSTEP / 8) : (uint32_t)(SH::NSTEP / 4);
#define OCT_RUN(ONEDIR, ALWAYS) \
    run_steps<SH, BLK, ONEDIR, ALWAYS, DEAD>(Sb, BT, tg, grp, c2c, t, P.rk, P.P16, P.Q16, P.dtr_mask, dead_lim, k4_begin, k4_end)
    if (onedir && T16 == 65536u) OCT_RUN(true, true);
    else if (onedir)             OCT_RUN(true, false);
    else if constexpr (BLK != kBlkSync) OCT_RUN(false, false);
#undef OCT_RUN
    // every variant of run_steps ends with a group barrier: the entries are final here

    // ---- a7: stage-out (:164): whole packed words of the window ---------------------------------
    for (uint32_t idx = tg; idx < (uint32_t)(NW * NW); idx += G) {
        const uint32_t jw = idx / NW, iw = idx - jw * NW;
        if (DEAD && !(iw < ncol && jw < nrow)) continue;
        const uint32_t word = gather_word<SH>(S, iw, jw);
        P.lat[(size_t)((wy0 + jw) & LWm) * LW + ((wx0 + iw) & LWm)] = word;
        net -= x_moment(word, iw);
    }

    // counters: net deposits (one atomic per warp) and the tracked height of site (0,0): the site west
    // of the row start is inactive in this launch, so the change of h(0,0) is twice the change of the
    // number of up-links between them
    if (has00) {
        d00 += row_links_up<SH>(Sb, x00, y00, tg);
        if (d00 != 0) atomicAdd(&P.counters[1], (unsigned long long)(long long)(2 * d00));
    }
    net = __reduce_add_sync(0xFFFFFFFFu, net);
    if ((threadIdx.x & 31) == 0 && net != 0) atomicAdd(&P.counters[0], (unsigned long long)(long long)net);
}

}  // namespace octb

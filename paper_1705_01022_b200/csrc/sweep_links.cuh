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
#include <type_traits>
#include <cuda_runtime.h>

#include "philox.cuh"
#include "sweep.cuh"

namespace octb {

constexpr uint32_t kEntryMin = 0x01000100u;   // (W,E,S,N) = (0,1,0,1): local minimum, Eq. (1)
constexpr uint32_t kEntryMax = 0x00010001u;   // (1,0,1,0): local maximum

// G_ = threads of the worker group that owns one domain: a multiple of 32 (one or several warps), or 16 -- two
// domains per warp, for domains with only 16 thread cells (TC=2,2 at D = 64: the paper's second production
// configuration, Fig. 5 :236-244).  DPB_ = domains per CTA.
template <int LOG2D, int TCX, int TCY, int G_, int DPB_>
struct LinkShape {
    static constexpr int D = 1 << LOG2D;
    static constexpr int CX = 4 << TCX, CY = 4 << TCY;
    static constexpr int NCX = D / CX, NCY = D / CY, NCELL = NCX * NCY;
    static constexpr int NSTEP = CX * CY;                 // collective steps per domain sweep (R12)
    static constexpr int G = G_, DPB = DPB_;              // threads per worker group (one domain), domains per CTA
    static constexpr int CPT = NCELL / G;                 // cells per thread per collective step
    static constexpr int NTHREADS = G * DPB;
    static constexpr int NW = D / 4 + 1;                  // window edge in packed words (halo included)
    static constexpr int P = 4 * NW;                      // entries per row (multiple of 4: 128-bit rows)
    static constexpr int ROWS = 4 * NW + 1;               // one spare row below row 0 for stray S-writes
    static constexpr int ENTRY_WORDS = ROWS * P;
    // block-step words (one per collective step, R13/R17) are kept in shared memory for BTW steps at a time; two
    // domains per warp keep 16 only, so that six CTAs of two domains fit one SM (6 x (2 x 18832 + 1024) B <= 228 KiB)
    static constexpr int BTW = (G_ == 16 && NSTEP > 64) ? 16 : (NSTEP < 64 ? NSTEP : 64);
    static constexpr int SMEM_PER_DOMAIN = (ENTRY_WORDS + BTW) * 4;
    static constexpr int SMEM_BYTES = SMEM_PER_DOMAIN * DPB;
    static_assert(LOG2D <= 7, "x and y are decoded in 8-bit fields: D + CX - 2 must stay below 256");
    static_assert(NCELL % G == 0 && CPT >= 1, "every thread carries the same number of cells");
    static_assert(G == 16 || G % 32 == 0, "a group is half a warp or whole warps");
    // one warp or half a warp per 64 x 64 domain: the fast staging path (each window word is loaded once, the east
    // halo bits come by shuffle, the north ones by shuffle or from the lane's own next word)
#ifndef OCT_LINKS_FAST_STAGE
#define OCT_LINKS_FAST_STAGE 1
#endif
    static constexpr bool FAST_17 = (OCT_LINKS_FAST_STAGE && (G == 32 || G == 16) && NW == 17);
    static_assert(CX <= D && CY <= D, "cell larger than domain");
};

// bits 0,2,4,6 of b -> bit 0 of bytes 0,1,2,3 (multiply-shift scatter; partial products never collide
// in a way that carries into a kept bit)
__device__ __forceinline__ uint32_t scatter4(uint32_t b) { return ((b & 0x55u) * 0x41041u) & 0x01010101u; }

// four entries of one site row from the scattered slope bytes: sx / sy = sigma_x / sigma_y of the four sites,
// sxe = sigma_x of their east neighbours, syn = sigma_y of their north neighbours (4 x 4 byte transpose by PRMT)
__device__ __forceinline__ uint4 entries_of_row(uint32_t sx, uint32_t sxe, uint32_t sy, uint32_t syn)
{
    const uint32_t t0 = __byte_perm(sx, sxe, 0x5140), t1 = __byte_perm(sx, sxe, 0x7362);
    const uint32_t u0 = __byte_perm(sy, syn, 0x5140), u1 = __byte_perm(sy, syn, 0x7362);
    uint4 q;
    q.x = __byte_perm(t0, u0, 0x5410); q.y = __byte_perm(t0, u0, 0x7632);
    q.z = __byte_perm(t1, u1, 0x5410); q.w = __byte_perm(t1, u1, 0x7632);
    return q;
}

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
        *reinterpret_cast<uint4*>(S + (4 * jw + j) * SH::P + 4 * iw) = entries_of_row(sx, sxe, sy[j], sy[j + 1]);
    }
}

// The same with the four site rows visited in the order (j + rot) & 3.  Used for the last window column, where the
// lanes hold consecutive word rows of ONE column: lane jw's 128-bit store of site row 4 jw + jj falls into bank
// group (4 jw + jj) mod 8 (pitch 4 * 17 words), so with rot = jw >> 1 eight consecutive lanes hit eight different groups.
template <class SH>
__device__ __forceinline__ void expand_word_rot(uint32_t* __restrict__ S, uint32_t iw, uint32_t jw, uint32_t A,
                                                uint32_t Ew, uint32_t Nw, uint32_t rot)
{
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint32_t jj = ((uint32_t)j + rot) & 3u;
        const uint32_t lo = __funnelshift_r(A, Nw, 8u * jj);               // (Nw:A) >> 8 jj: rows jj.. of A, then row 0 of Nw
        const uint32_t sx = scatter4(lo);
        const uint32_t sxe = (sx >> 8) | (((Ew >> (8u * jj)) & 1u) << 24);
        *reinterpret_cast<uint4*>(S + (4 * jw + jj) * SH::P + 4 * iw) = entries_of_row(sx, sxe, scatter4(lo >> 1), scatter4(lo >> 9));
    }
}

// own links (bytes 0 and 2) of the four entries of one site row -> the row's 8 bits of the packed word
__device__ __forceinline__ uint32_t row_bits(const uint4 q)
{
    const uint32_t z = q.x + 4u * q.y + 16u * q.z + 64u * q.w;           // W bits at 0,2,4,6; S bits at 16,18,20,22
    return (z & 0x55u) | ((z >> 15) & 0xAAu);
}

// Gather the own links of 16 entries back into one packed word.
template <class SH>
__device__ __forceinline__ uint32_t gather_word(const uint32_t* __restrict__ S, uint32_t iw, uint32_t jw)
{
    uint32_t word = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j)
        word |= row_bits(*reinterpret_cast<const uint4*>(S + (4 * jw + j) * SH::P + 4 * iw)) << (8 * j);
    return word;
}

template <class SH>
__device__ __forceinline__ uint32_t gather_word_rot(const uint32_t* __restrict__ S, uint32_t iw, uint32_t jw, uint32_t rot)
{
    uint32_t word = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint32_t jj = ((uint32_t)j + rot) & 3u;
        word |= row_bits(*reinterpret_cast<const uint4*>(S + (4 * jw + jj) * SH::P + 4 * iw)) << (8u * jj);
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

// synchronise the worker group of one domain.  Groups of at most one warp: __syncwarp over the warp's live lanes
// (wmask; with G = 16 the two domains of a warp step together); one group per CTA: the CTA barrier; else a named barrier.
template <int G, int DPB>
__device__ __forceinline__ void links_sync(int grp, uint32_t wmask)
{
    if constexpr (G <= 32) {
        __syncwarp(wmask);
    } else if constexpr (DPB == 1) {
        __syncthreads();
    } else {
        asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "n"(G) : "memory");
    }
}

#ifndef OCT_LINKS_MERGE
#define OCT_LINKS_MERGE 0     // 0: every cell slot of a lane issues its own group of five stores (round 1)
#endif

// flip_links under a predicate, as five predicated stores (no branch: the merged store group below must stay
// straight-line code, a divergent branch per step costs more than the stores it would skip)
template <class SH>
__device__ __forceinline__ void flip_links_if(bool on, uint32_t* Sb, uint32_t i, bool up)
{
    const uint32_t a = (uint32_t)__cvta_generic_to_shared(Sb + i);
    const uint32_t e = up ? kEntryMax : kEntryMin, v1 = up ? 1u : 0u, v0 = up ? 0u : 1u;
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %0, 0;\n\t"
        "@p st.shared.u32 [%1], %2;\n\t"
        "@p st.shared.u8 [%1+-3], %3;\n\t"          // west neighbour's E link
        "@p st.shared.u8 [%1+4], %4;\n\t"           // east neighbour's W link
        "@p st.shared.u8 [%1+%5], %3;\n\t"          // south neighbour's N link
        "@p st.shared.u8 [%1+%6], %4;\n\t}"         // north neighbour's S link
        :: "r"((uint32_t)on), "r"(a), "r"(e), "r"(v1), "r"(v0), "n"(-4 * SH::P + 3), "n"(4 * SH::P + 2) : "memory");
}

// Carry out the decisions of one collective step.  With two cells per lane the accepted updates are spread thinly
// (about 6 of 32 lanes per cell slot, and every store instruction costs a shared-memory wavefront or more however few
// lanes take part), so the two slots are merged into ONE group of five stores: a lane with two accepted updates hands
// its second one to lane ^ 16 if that lane has none (one shuffle); what is left over -- both lanes busy, seldom --
// goes in a second, warp-uniformly skipped group.  Which lane performs a store does not matter: the updates of a
// phase touch disjoint links (R15/R16).
template <class SH, bool ONEDIR, bool ALWAYS, int CPT>
__device__ __forceinline__ void apply_step(const Rule<ONEDIR, ALWAYS>& rule, uint32_t* Sb, const uint32_t (&idx)[CPT], const int (&dec)[CPT],
                                           uint32_t wmask)
{
    if constexpr (OCT_LINKS_MERGE && CPT == 2 && SH::G >= 32) {
        const bool a0 = dec[0] != 0, a1 = dec[1] != 0;
        const bool two = a0 && a1, none = !(a0 || a1);
        uint32_t offer = idx[1] | (two ? 0x80000000u : 0u) | (none ? 0x40000000u : 0u);
        if constexpr (!ONEDIR) offer |= dec[1] > 0 ? 0x20000000u : 0u;
        const uint32_t got = __shfl_xor_sync(0xFFFFFFFFu, offer, 16);
        const bool take = none && (got >> 31);                 // the partner's second update is carried out here
        const bool given = two && ((got >> 30) & 1u);          // ... and this lane's second one over there
        const uint32_t i1 = take ? (got & 0xFFFFu) : (a0 ? idx[0] : idx[1]);
        bool up1 = rule.dep, up2 = rule.dep;
        if constexpr (!ONEDIR) { up1 = take ? (got & 0x20000000u) != 0u : (a0 ? dec[0] > 0 : dec[1] > 0); up2 = dec[1] > 0; }
        flip_links_if<SH>(a0 || a1 || take, Sb, i1, up1);
        const bool rest = two && !given;
        if (__any_sync(0xFFFFFFFFu, rest)) flip_links_if<SH>(rest, Sb, idx[1], up2);
    } else {
#pragma unroll
        for (int j = 0; j < CPT; ++j) rule.template apply<SH>(Sb, idx[j], dec[j]);
    }
}

// The collective single-hit steps of one domain sweep (:168-174).
// DEAD: dead-border device layer (:135): attempts whose domain-local x or y is >= dead_lim are not carried out.
template <class SH, int BLK, bool ONEDIR, bool ALWAYS, bool DEAD>
__device__ __forceinline__ void run_steps(uint32_t* __restrict__ Sb, uint32_t* __restrict__ BT, uint32_t tg, int grp, uint32_t wmask,
                                         uint32_t c2b, uint32_t c2c, uint32_t t, const PhiloxRoundKeys& rk, uint32_t P16, uint32_t Q16, uint32_t dtr_mask,
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
    constexpr int kUnrollK4 = CPT >= 4 ? 2 : (SH::BTW / 4 < 8 / CPT ? SH::BTW / 4 : 8 / CPT);
    constexpr uint32_t RB = SH::BTW / 4;             // groups of four steps per fill of the block-step ring
#pragma unroll 1
    for (uint32_t kb = k4_begin; kb < k4_end; kb += RB) {
    // ---- a3: block-step words of the next BTW steps (:170, :172; R13/R17/R24); the previous step ended with a barrier
    for (uint32_t q = tg; q < RB && kb + q < k4_end; q += G) {
        uint32_t o[4];
        philox4x32_10(kb + q, 0u, c2b, t, rk, o);
        *reinterpret_cast<uint4*>(BT + 4 * q) = make_uint4(o[0], o[1], o[2], o[3]);
    }
    links_sync<G, SH::DPB>(grp, wmask);
    const uint32_t ke = kb + RB < k4_end ? kb + RB : k4_end;
#pragma unroll kUnrollK4
    for (uint32_t k4 = kb; k4 < ke; ++k4) {
        uint32_t rw[CPT][4];
#pragma unroll
        for (int j = 0; j < CPT; ++j) philox4x32_10(k4, tg + j * G, c2c, t, rk, rw[j]);

        const uint4 bq = *reinterpret_cast<const uint4*>(BT + 4 * (k4 - kb));   // one broadcast load for four steps
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
                links_sync<G, SH::DPB>(grp, wmask);
                apply_step<SH>(rule, Sb, idx, dec, wmask);
                links_sync<G, SH::DPB>(grp, wmask);
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
                    links_sync<G, SH::DPB>(grp, wmask);
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
                apply_step<SH>(rule, Sb, idx, dec, wmask);
                links_sync<G, SH::DPB>(grp, wmask);
            }
        }
    }
    }
}

// number of set W links of the sites (0..n00-1, y00) of the domain: with n00 = x00 + 1 it is h(x00,y00) minus the
// height of the inactive site west of the row start, up to a constant (used before and after the sweep, R20)
template <class SH>
__device__ __forceinline__ int row_links_up(const uint32_t* Sb, uint32_t n00, uint32_t y00, uint32_t tg)
{
    int n = 0;
    for (uint32_t x = tg; x < n00; x += SH::G) n += (int)(Sb[y00 * SH::P + x] & 1u);
    return n;
}

__device__ __forceinline__ const SweepParams& common_params(const SweepParams& p) { return p; }
__device__ __forceinline__ const SweepParams& common_params(const SweepBatchParams& p) { return p.common; }

// DEAD = false: tiled device layers DTr / DT (four launches per MCS, one per domain set);
// DEAD = true : dead-border device layers DB / cDB / DBh (all tiles in one launch; the rim of width dead_w is
//               never updated, and words shared with the next tile are neither read, counted nor written, :166).
template <int LOG2D, int TCX, int TCY, int BLK, int G_, int DPB, bool DEAD, bool BATCH = false>
__global__ void __launch_bounds__(LinkShape<LOG2D, TCX, TCY, G_, DPB>::NTHREADS)
sweep_links_kernel(const __grid_constant__ typename std::conditional<BATCH, SweepBatchParams, SweepParams>::type PP)
{
    using SH = LinkShape<LOG2D, TCX, TCY, G_, DPB>;
    constexpr int D = SH::D, G = SH::G, NW = SH::NW;

    extern __shared__ __align__(16) uint32_t smem_raw[];
    const int grp = threadIdx.x / G;                 // worker group inside the CTA
    const uint32_t tg = threadIdx.x % G;             // thread inside the group
    uint32_t* S0 = smem_raw + grp * (SH::SMEM_PER_DOMAIN / 4);
    uint32_t* S = S0 + SH::P;                        // row 0 of the window (one spare row below it)
    uint32_t* BT = S0 + SH::ENTRY_WORDS;             // block-step words of this domain sweep

    // one lattice: everything comes from the parameter block (the round keys stay in the constant bank);
    // batch: blockIdx.y picks the member; its key schedule is rebuilt from its seed (registers)
    const SweepParams& P = common_params(PP);
    uint32_t* __restrict__ lat;
    unsigned long long* counters;
    uint32_t t;
    PhiloxRoundKeys rk_member;
    if constexpr (BATCH) {
        const BatchMember& mb = PP.m[blockIdx.y];
        lat = mb.lat; counters = mb.counters; t = mb.t;
#pragma unroll
        for (int r = 0; r < 10; ++r) { rk_member.k0[r] = mb.seed_lo + (uint32_t)r * 0x9E3779B9u; rk_member.k1[r] = mb.seed_hi + (uint32_t)r * 0xBB67AE85u; }
    } else {
        lat = P.lat; counters = P.counters; t = P.t;
    }
    const PhiloxRoundKeys& rk = BATCH ? rk_member : P.rk;      // compile-time choice
    const uint32_t L = P.L, Lm = L - 1u;

    const uint32_t dom = blockIdx.x * DPB + grp;
    // the live lanes of this warp: a whole group leaves together (G = 16: half a warp may leave)
    const uint32_t wmask = G <= 32 ? __ballot_sync(0xFFFFFFFFu, dom < P.ndom) : 0xFFFFFFFFu;
    if (dom >= P.ndom) return;

    // ---- a1: per-MCS control from the global stream (:144, :150; R10) --------------------------
    uint32_t Gw[4];                                  // dead-border layers: this launch is interval P.si of the sweep (R27)
    philox4x32_10(DEAD ? P.si : 0u, 0u, kTagGlobal << 30, t, rk, Gw);
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
        set = P.si;
        const uint32_t lnt = P.log2L - LOG2D;
        const uint32_t I = dom & ((1u << lnt) - 1u), J = dom >> lnt;
        gx = (Ox + (I << LOG2D)) & Lm;
        gy = (Oy + (J << LOG2D)) & Lm;
        dead_w = P.dead_w;                                              // :166, R22/R28
    }
    const uint32_t offx = gx & 3u, offy = gy & 3u;
    const uint32_t LW = L >> 2, LWm = LW - 1u, wx0 = gx >> 2, wy0 = gy >> 2;
    uint32_t* Sb = S + offy * SH::P + offx;          // entry of the domain's site (0,0)
    // window words this domain reads, counts and writes back: all of them, or (dead border) only those that hold no
    // site of the next tile -- the last active site's E / N links still lie inside them (:166).  The other words
    // belong to the next tile, which writes them in this same launch: they are not even loaded (zeros stand in;
    // they only reach entries of dead sites, which are never tested).
    const uint32_t ncol = DEAD ? ((offx + (uint32_t)D - dead_w) >> 2) + 1u : (uint32_t)NW;
    const uint32_t nrow = DEAD ? ((offy + (uint32_t)D - dead_w) >> 2) + 1u : (uint32_t)NW;
    auto kept = [&](uint32_t iw, uint32_t jw) -> bool { return !DEAD || (iw < ncol && jw < nrow); };
    auto word_ptr = [&](uint32_t iw, uint32_t jw) -> uint32_t* { return lat + (size_t)((wy0 + jw) & LWm) * LW + ((wx0 + iw) & LWm); };
    auto put_word = [&](uint32_t iw, uint32_t jw, uint32_t word) {
        if constexpr (DEAD) store_tile_word(word_ptr(iw, jw), word, iw, jw, offx, offy, (uint32_t)D, dead_w);
        else *word_ptr(iw, jw) = word;
    };

    // Programmatic dependent launch: the launches of one MCS depend on each other (kernel boundary = the device-wide
    // synchronisation of :144), but everything above touches no global memory, so the next launch's CTAs may take
    // their SM slots while this grid drains and wait HERE for its completion (hides the launch ramp: matters for
    // small lattices / ensembles, where a launch lasts ~20 us).
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");

    // ---- a2: stage-in (:164): packed words -> link entries -------------------------------------
    int net = 0;                                     // deposits - removals, from the x-moments (see x_moment)
    if constexpr (SH::FAST_17 && G == 16) {
        // Half a warp, window of 17 x 17 words: lane iw holds column iw of all 17 word rows (and lane jw word (16, jw)
        // of the last column; lane 0 also (16, 16)).  Every word is loaded ONCE, all loads in flight together: the east
        // word is the next lane's (shuffle inside the half warp), the north word the lane's own next register.
        const uint32_t iw = tg;
        uint32_t A[NW + 1], C, C16;
#pragma unroll
        for (int jw = 0; jw < NW; ++jw) A[jw] = kept(iw, jw) ? *word_ptr(iw, jw) : 0u;
        A[NW] = 0u;
        C = kept(NW - 1, tg) ? *word_ptr(NW - 1, tg) : 0u;
        C16 = (tg == 0u && kept(NW - 1, NW - 1)) ? *word_ptr(NW - 1, NW - 1) : 0u;
#pragma unroll
        for (int jw = 0; jw < NW; ++jw) {
            const uint32_t e1 = __shfl_down_sync(wmask, A[jw], 1, 16);
            const uint32_t e2 = jw < 16 ? __shfl_sync(wmask, C, jw, 16) : __shfl_sync(wmask, C16, 0, 16);
            expand_word<SH>(S, iw, jw, A[jw], iw == 15u ? e2 : e1, A[jw + 1]);
            if (kept(iw, jw)) net += x_moment(A[jw], iw);
        }
        // last column: lane jw expands word (16, jw), lane 0 then (16, 16); its north word is the next lane's
        const uint32_t Cn = __shfl_down_sync(wmask, C, 1, 16), Cn15 = __shfl_sync(wmask, C16, 0, 16);
        expand_word_rot<SH>(S, NW - 1, tg, C, 0u, tg == 15u ? Cn15 : Cn, tg >> 1);
        if (kept(NW - 1, tg)) net += x_moment(C, NW - 1);
        if (tg == 0u) {
            expand_word<SH>(S, NW - 1, NW - 1, C16, 0u, 0u);
            if (kept(NW - 1, NW - 1)) net += x_moment(C16, NW - 1);
        }
    } else if constexpr (SH::FAST_17) {
        // One warp, window of 17 x 17 words.  Lanes 0-15 take the 16 leading words of an even word row, lanes 16-31 of
        // the odd row above it, nine row pairs in all; lanes 0-16 then take the last column.  Every word is loaded
        // ONCE: the east word is the next lane's (or the last column's), the north word the partner lane's (^16).
        // Each 128-bit store of a quarter warp covers 128 contiguous bytes: no bank conflicts.
        constexpr int NP = (NW + 1) / 2;             // row pairs
        const uint32_t hi = tg >> 4, iw = tg & 15u;
        uint32_t A[NP + 1], C;
#pragma unroll
        for (int it = 0; it < NP; ++it) {
            const uint32_t jw = 2u * it + hi;
            A[it] = (jw < (uint32_t)NW && kept(iw, jw)) ? *word_ptr(iw, jw) : 0u;
        }
        A[NP] = 0u;
        C = (tg < (uint32_t)NW && kept(NW - 1, tg)) ? *word_ptr(NW - 1, tg) : 0u;
#pragma unroll
        for (int it = 0; it < NP; ++it) {
            const uint32_t jw = 2u * it + hi;
            const uint32_t e1 = __shfl_down_sync(0xFFFFFFFFu, A[it], 1), e2 = __shfl_sync(0xFFFFFFFFu, C, jw);
            const uint32_t Nw = __shfl_xor_sync(0xFFFFFFFFu, hi ? A[it] : A[it + 1], 16);
            if (jw < (uint32_t)NW) {
                expand_word<SH>(S, iw, jw, A[it], iw == 15u ? e2 : e1, Nw);
                if (kept(iw, jw)) net += x_moment(A[it], iw);
            }
        }
        const uint32_t Cn = __shfl_down_sync(0xFFFFFFFFu, C, 1);
        if (tg < (uint32_t)NW) {
            expand_word_rot<SH>(S, NW - 1, tg, C, 0u, Cn, tg >> 1);       // the east links of this column are never read
            if (kept(NW - 1, tg)) net += x_moment(C, NW - 1);
        }
    } else {
        constexpr int NIT = (NW * NW + G - 1) / G;   // words per thread; loaded in chunks, all loads of a chunk before its first use
        constexpr int NCH = (NIT + 19) / 20, CH = (NIT + NCH - 1) / NCH;    // at most 20 words (60 loads) per thread in flight
#pragma unroll 1
        for (int c0 = 0; c0 < NIT; c0 += CH) {
            uint32_t A[CH], Ew[CH], Nw[CH];
#pragma unroll
            for (int it = 0; it < CH; ++it) {
                const uint32_t idx = tg + (c0 + it) * G;
                A[it] = Ew[it] = Nw[it] = 0u;
                if (idx < (uint32_t)(NW * NW)) {
                    const uint32_t jw = idx / NW, iw = idx - jw * NW;
                    if constexpr (DEAD) {
                        if (kept(iw, jw)) A[it] = *word_ptr(iw, jw);
                        if (kept(iw + 1, jw)) Ew[it] = *word_ptr(iw + 1, jw);
                        if (kept(iw, jw + 1)) Nw[it] = *word_ptr(iw, jw + 1);
                    } else {                          // words east / north of the window are read but never used
                        A[it] = *word_ptr(iw, jw); Ew[it] = *word_ptr(iw + 1, jw); Nw[it] = *word_ptr(iw, jw + 1);
                    }
                }
            }
#pragma unroll
            for (int it = 0; it < CH; ++it) {
                const uint32_t idx = tg + (c0 + it) * G;
                if (idx < (uint32_t)(NW * NW)) {
                    const uint32_t jw = idx / NW, iw = idx - jw * NW;
                    expand_word<SH>(S, iw, jw, A[it], Ew[it], Nw[it]);
                    if (kept(iw, jw)) net += x_moment(A[it], iw);
                }
            }
        }
    }
    const uint32_t c2b = (kTagBlock << 30) | (set << 28) | dom, c2c = (kTagCell << 30) | (set << 28) | dom;
    links_sync<G, DPB>(grp, wmask);

    // is the lattice origin (0,0) an active site of this domain?  (anchor tracking, R20)
    const uint32_t x00 = (0u - gx) & Lm, y00 = (0u - gy) & Lm;
    const bool has00 = x00 < (uint32_t)D && y00 < (uint32_t)D;
    const uint32_t n00 = has00 ? x00 + 1u : 0u, r00 = has00 ? y00 : 0u;
    int d00 = -row_links_up<SH>(Sb, n00, r00, tg);
    links_sync<G, DPB>(grp, wmask);                  // the first phase may write at once

    // ---- a4-a6: collective single-hit steps (:168) ---------------------------------------------
    // launch-uniform specialisation of the acceptance rule (the sync variant is only used with p*q = 0, R16)
    const bool onedir = BLK == kBlkSync || P.P16 == 0u || P.Q16 == 0u;
    const uint32_t T16 = P.Q16 == 0u ? P.P16 : P.Q16;
    const uint32_t dead_lim = (uint32_t)D - dead_w;
    const uint32_t k4_per = DEAD ? (uint32_t)(SH::NSTEP / 4) >> P.ka : (uint32_t)(SH::NSTEP / 4);   // steps of this interval
    const uint32_t k4_begin = DEAD ? P.si * k4_per : 0u, k4_end = k4_begin + k4_per;
#define OCT_RUN(ONEDIR, ALWAYS) \
    run_steps<SH, BLK, ONEDIR, ALWAYS, DEAD>(Sb, BT, tg, grp, wmask, c2b, c2c, t, rk, P.P16, P.Q16, P.dtr_mask, dead_lim, k4_begin, k4_end)
    if (onedir && T16 == 65536u) OCT_RUN(true, true);
    else if (onedir)             OCT_RUN(true, false);
    else if constexpr (BLK != kBlkSync) OCT_RUN(false, false);
#undef OCT_RUN
    // every variant of run_steps ends with a group barrier: the entries are final here

    // ---- a7: stage-out (:164): whole packed words of the window ---------------------------------
    if constexpr (SH::FAST_17 && G == 16) {
        const uint32_t iw = tg;
#pragma unroll 4
        for (uint32_t jw = 0; jw < (uint32_t)NW; ++jw) {
            if (!kept(iw, jw)) continue;
            const uint32_t word = gather_word<SH>(S, iw, jw);
            put_word(iw, jw, word);
            net -= x_moment(word, iw);
        }
        if (kept(NW - 1, tg)) {
            const uint32_t word = gather_word_rot<SH>(S, NW - 1, tg, tg >> 1);
            put_word(NW - 1, tg, word);
            net -= x_moment(word, NW - 1);
        }
        if (tg == 0u && kept(NW - 1, NW - 1)) {
            const uint32_t word = gather_word<SH>(S, NW - 1, NW - 1);
            put_word(NW - 1, NW - 1, word);
            net -= x_moment(word, NW - 1);
        }
    } else if constexpr (SH::FAST_17) {
        const uint32_t hi = tg >> 4, iw = tg & 15u;
#pragma unroll 3
        for (uint32_t jw = hi; jw < (uint32_t)NW; jw += 2) {
            if (!kept(iw, jw)) continue;
            const uint32_t word = gather_word<SH>(S, iw, jw);
            put_word(iw, jw, word);
            net -= x_moment(word, iw);
        }
        if (tg < (uint32_t)NW && kept(NW - 1, tg)) {
            const uint32_t word = gather_word_rot<SH>(S, NW - 1, tg, tg >> 1);
            put_word(NW - 1, tg, word);
            net -= x_moment(word, NW - 1);
        }
    } else {
        for (uint32_t idx = tg; idx < (uint32_t)(NW * NW); idx += G) {
            const uint32_t jw = idx / NW, iw = idx - jw * NW;
            if (!kept(iw, jw)) continue;
            const uint32_t word = gather_word<SH>(S, iw, jw);
            put_word(iw, jw, word);
            net -= x_moment(word, iw);
        }
    }

    // counters: net deposits (one atomic per warp) and the tracked height of site (0,0): the site west
    // of the row start is inactive in this launch, so the change of h(0,0) is twice the change of the
    // number of up-links between them
    d00 += row_links_up<SH>(Sb, n00, r00, tg);
    if (d00 != 0) atomicAdd(&counters[1], (unsigned long long)(long long)(2 * d00));
    net = __reduce_add_sync(wmask, net);
    if ((threadIdx.x & 31) == 0 && net != 0) atomicAdd(&counters[0], (unsigned long long)(long long)net);
}

}  // namespace octb

// Sweep kernel, link-entry layout: one launch = one domain-set sweep of any device-layer scheme of
// arXiv 1705.01022 (DTr / DT: Sec. 3.0.2-3.0.3; DB / cDB / DBh: Sec. 3.0.1, :133-140, :166)
// with any of the single-hit block layers (Sec. 3.1, :168-174), for device-layer domains of D <= 256 sites (D = 256 with
// two-byte entries only: four-byte entries of a 256 x 256 domain do not fit shared memory).
//
// Why a second layout (profiles/r3_sweep.md, last section): on the bit-packed window the update test costs ~115 SASS
// instructions per attempt, almost all of them shift/mask arithmetic and shared-memory atomics, and the
// ALU pipe binds.  Here the window is unpacked ONCE per domain sweep into one 32-bit *entry* per site that
// carries the four links of that site, one byte each (0x00 = slope -1, 0xFF = slope +1):
//      byte 0  W = sigma_x(x,y)     byte 1  E = sigma_x(x+1,y)
//      byte 2  S = sigma_y(x,y)     byte 3  N = sigma_y(x,y+1)                      (:140, R3)
// so that
//   * the eligibility test of Eq. (1) (:27-34) is one LDS.32 and one compare: local minimum
//     (W,E,S,N) = (0,1,0,1) <=> entry == 0xFF00FF00, local maximum <=> entry == 0x00FF00FF;
//   * an accepted update is five plain stores: the site's own entry and one byte in each of the four
//     neighbouring entries (every link is stored twice, once per end site).  No atomics are needed:
//     a link can only be changed by an update at one of its two end sites, two nearest-neighbour sites
//     are never updated in the same phase (:174, R15/R16), and byte stores leave the other bytes of a
//     word alone.  Entries of sites outside the active D x D square (halo and alignment padding) take
//     stray byte writes in their E/N bytes only, which are never read and never written back.
//   * the window is kept in the lattice's own 4-site word alignment (pitch D+4 entries), so stage-in
//     expands a packed word into four 128-bit stores and stage-out gathers it back from four 128-bit
//     loads.  Both are byte permutes (profiles/r2_sweep.md: the kernel is bound by the instruction issue
//     rate at three warps per scheduler, and staging was 39 % of its instructions): a link byte is the
//     SIGN-REPLICATED top bit of a byte of a shifted copy of the packed word (PRMT with selector bit 3),
//     12 shifts + 24 permutes per 16 entries; the way back is 2 permutes, 2 masks and one multiply per row.
// Everything else (Philox streams, per-MCS control, cell geometry, phases) is as in sweep.cuh and
// follows the same readings R10-R19 of DESIGN.md.
#pragma once
#include <cstdint>
#include <type_traits>
#include <cuda_runtime.h>

#include "philox.cuh"
#include "sweep.cuh"

namespace octb {

constexpr uint32_t kEntryMin = 0xFF00FF00u;   // (W,E,S,N) = (0,1,0,1): local minimum, Eq. (1); a set link is the byte 0xFF
constexpr uint32_t kEntryMax = 0x00FF00FFu;   // (1,0,1,0): local maximum
// Two-byte entries (EB = 2): a site keeps only its OWN links (W, S); the test gathers (W, S, E, N) from three loads --
// the entry, the east neighbour's W byte, the north neighbour's S byte -- and an update is three stores.  Half the shared
// memory per domain, i.e. twice the domains in flight: for shapes with few cells per domain (TC=2,2: 16 cells per 64 x 64
// domain), which are bound by the latency of the step chain, not by the shared-memory pipe (profiles/r2_sweep.md).
constexpr uint32_t kEntry2Min = 0xFFFF0000u;  // (W,S,E,N) = (0,0,1,1)
constexpr uint32_t kEntry2Max = 0x0000FFFFu;

// G_ = threads of the worker group that owns one domain: a multiple of 32 (one or several warps), or 16 -- two
// domains per warp, for domains with only 16 thread cells (TC=2,2 at D = 64: the paper's second production
// configuration, Fig. 5 :236-244).  DPB_ = domains per CTA.
template <int LOG2D, int TCX, int TCY, int G_, int DPB_, int EB_ = 4>
struct LinkShape {
    static constexpr int EB = EB_;                        // bytes per entry: 4 (W,E,S,N) or 2 (W,S)
    static_assert(EB == 4 || EB == 2, "entries are four or two link bytes");
    static constexpr int D = 1 << LOG2D;
    static constexpr int CX = 4 << TCX, CY = 4 << TCY;
    static constexpr int NCX = D / CX, NCY = D / CY, NCELL = NCX * NCY;
    static constexpr int NSTEP = CX * CY;                 // collective steps per domain sweep (R12)
    static constexpr int G = G_, DPB = DPB_;              // threads per worker group (one domain), domains per CTA
    static constexpr int CPT = NCELL / G;                 // cells per thread per collective step
    static constexpr int NTHREADS = G * DPB;
    static constexpr int NW = D / 4 + 1;                  // window edge in packed words (halo included)
    static constexpr int P = 4 * NW;                      // entries per row (multiple of 4: 128-bit rows)
    static constexpr int ROWS = EB == 4 ? 4 * NW + 1 : 4 * NW;   // four-byte entries: one spare row below row 0 for stray S-writes
    static constexpr int ENTRY_WORDS = ROWS * P * EB / 4;
    // block-step words (one per collective step, R13/R17) are kept in shared memory for BTW steps at a time; two
    // domains per warp keep 16 only, so that six CTAs of two domains fit one SM (6 x (2 x 18832 + 1024) B <= 228 KiB)
    static constexpr int BTW = (G_ == 16 && NSTEP > 64) ? 16 : (NSTEP < 64 ? NSTEP : 64);
    static constexpr int SMEM_PER_DOMAIN = (ENTRY_WORDS + BTW) * 4;
    static constexpr int SMEM_BYTES = SMEM_PER_DOMAIN * DPB;
    // x and y of a site travel in one register: 8-bit fields (x | y << 8) while D + CX - 2 stays below 256, 16-bit fields
    // (x | y << 16) for D = 256 -- two-byte entries only: a 256 x 256 window of four-byte entries does not fit shared memory
    static constexpr bool WIDE = LOG2D == 8;
    static constexpr int YSH = WIDE ? 16 : 8;
    static_assert(LOG2D <= 7 || (LOG2D == 8 && EB == 2), "D = 256 needs two-byte entries");
    static_assert(NCELL % G == 0 && CPT >= 1, "every thread carries the same number of cells");
    static_assert(G == 16 || G % 32 == 0, "a group is half a warp or whole warps");
    // one warp or half a warp per 64 x 64 domain: the fast staging path (each window word is loaded once, the east
    // halo bits come by shuffle, the north ones by shuffle or from the lane's own next word)
#ifndef OCT_LINKS_FAST_STAGE
#define OCT_LINKS_FAST_STAGE 1
#endif
    static constexpr bool FAST_17 = (OCT_LINKS_FAST_STAGE && (G == 32 || G == 16) && NW == 17);
    static_assert(ENTRY_WORDS % 4 == 0, "the block-step ring behind the entries is read with 128-bit loads");
    static_assert(CX <= D && CY <= D, "cell larger than domain");
};

// byte permute with the full 4-bit selectors of PTX prmt: selector nibble n picks byte (n & 7) of {a, b}; n & 8 replicates
// that byte's top bit over the whole result byte (0x00 / 0xFF)
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel)
{
    uint32_t d;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));
    return d;
}

// Expand packed word A (with its east neighbour Ew and north neighbour Nw) into 16 entries.
// Shifted copies of A put one link bit of every site row at the top of that row's byte: sigma_x of site i at the top
// of the bytes of A << (7 - 2i), sigma_y of site i at the top of the bytes of A << (6 - 2i); sign-replicating permutes
// then write the link bytes straight into place: (W,E) pairs of two rows from one permute, then one permute per entry.
template <class SH>
__device__ __forceinline__ void expand_word(uint32_t* __restrict__ S, uint32_t iw, uint32_t jw, uint32_t A,
                                            uint32_t Ew, uint32_t Nw)
{
    if constexpr (SH::EB == 2) {
        // two-byte entries: the 8 bytes of a site row are its 8 packed bits in order (W0, S0, W1, S1, ...), sign-replicated
        // from shifted copies: bit k of every row at the top of the bytes of A << (7 - k); no neighbour words needed
        uint32_t T[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) T[k] = A << (7 - k);
        uint32_t p01[4], p23[4];                                  // bits (2q, 2q+1) of rows 0, 1 / rows 2, 3
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            p01[q] = prmt(T[2 * q], T[2 * q + 1], 0xD9C8u);
            p23[q] = prmt(T[2 * q], T[2 * q + 1], 0xFBEAu);
        }
        unsigned short* E = reinterpret_cast<unsigned short*>(S);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t (&pp)[4] = j < 2 ? p01 : p23;
            const uint32_t sel = (j & 1) ? 0x7632u : 0x5410u;
            *reinterpret_cast<uint2*>(E + (4 * jw + j) * SH::P + 4 * iw) = make_uint2(prmt(pp[0], pp[1], sel), prmt(pp[2], pp[3], sel));
        }
        return;
    }
    uint32_t BW[5], BS[4], BN[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        BW[i] = A << (7 - 2 * i);                                 // byte j, top bit: sigma_x(site i, row j)
        BS[i] = A << (6 - 2 * i);                                 //                  sigma_y(site i, row j)
        BN[i] = __funnelshift_r(A, Nw, 18 + 2 * i);               // byte 0: sigma_y(site i, row 3); byte 1: sigma_y(site i, row 0 of Nw)
    }
    BW[4] = Ew << 7;                                              // sigma_x of the east word's site 0
    uint32_t e[4][4];                                             // e[j][i]: entry of site i of row j
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const uint32_t we01 = prmt(BW[i], BW[i + 1], 0xD9C8u);    // (W, E) of rows 0 and 1
        const uint32_t we23 = prmt(BW[i], BW[i + 1], 0xFBEAu);    // (W, E) of rows 2 and 3
        e[0][i] = prmt(we01, BS[i], 0xDC10u);                     // S = row 0, N = row 1 of sigma_y
        e[1][i] = prmt(we01, BS[i], 0xED32u);
        e[2][i] = prmt(we23, BS[i], 0xFE10u);
        e[3][i] = prmt(we23, BN[i], 0xDC32u);                     // N from the north word
    }
#pragma unroll
    for (int j = 0; j < 4; ++j)
        *reinterpret_cast<uint4*>(S + (4 * jw + j) * SH::P + 4 * iw) = make_uint4(e[j][0], e[j][1], e[j][2], e[j][3]);
}

// The same with the four site rows visited in the order (j + rot) & 3.  Used for the last window column, where the
// lanes hold consecutive word rows of ONE column: lane jw's 128-bit store of site row 4 jw + jj falls into bank
// group (4 jw + jj) mod 8 (pitch 4 * 17 words), so with rot = jw >> 1 eight consecutive lanes hit eight different groups.
template <class SH>
__device__ __forceinline__ void expand_word_rot(uint32_t* __restrict__ S, uint32_t iw, uint32_t jw, uint32_t A,
                                                uint32_t Ew, uint32_t Nw, uint32_t rot)
{
    if constexpr (SH::EB == 2) { expand_word<SH>(S, iw, jw, A, Ew, Nw); return; }   // (one word in 17: the conflicts do not matter)
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint32_t jj = ((uint32_t)j + rot) & 3u;
        const uint32_t lo = __funnelshift_r(A, Nw, 8u * jj);      // byte 0: row jj, byte 1: the row north of it
        const uint32_t le = (Ew >> (8u * jj)) << 7;               // byte 0, top bit: sigma_x of the east word's site 0 in row jj
        uint32_t q[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const uint32_t we = prmt(lo << (7 - 2 * i), i < 3 ? lo << ((5 - 2 * i) & 31) : le, 0x00C8u);
            q[i] = prmt(we, lo << (6 - 2 * i), 0xDC10u);
        }
        *reinterpret_cast<uint4*>(S + (4 * jw + jj) * SH::P + 4 * iw) = make_uint4(q[0], q[1], q[2], q[3]);
    }
}

// own links (bytes 0 and 2) of the four entries of one site row -> the row's 8 bits of the packed word, in the TOP byte
// of the result: two permutes line the eight link bytes up, two masks keep one distinct bit of each, and a multiply
// adds the four bytes (no carries: the bits are distinct)
__device__ __forceinline__ uint32_t row_bits_top(const uint4 q)
{
    const uint32_t t01 = prmt(q.x, q.y, 0x6240u);                 // (W0, W1, S0, S1)
    const uint32_t t23 = prmt(q.z, q.w, 0x6240u);                 // (W2, W3, S2, S3)
    return ((t01 & 0x08020401u) | (t23 & 0x80204010u)) * 0x01010101u;
}

// Gather the own links of 16 entries back into one packed word.
template <class SH>
__device__ __forceinline__ uint32_t gather_word(const uint32_t* __restrict__ S, uint32_t iw, uint32_t jw)
{
    uint32_t p[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        if constexpr (SH::EB == 2) {
            const uint2 v = *reinterpret_cast<const uint2*>(reinterpret_cast<const unsigned short*>(S) + (4 * jw + j) * SH::P + 4 * iw);
            p[j] = ((v.x & 0x08040201u) | (v.y & 0x80402010u)) * 0x01010101u;   // byte k keeps bit k; the multiply adds the bytes
        } else {
            p[j] = row_bits_top(*reinterpret_cast<const uint4*>(S + (4 * jw + j) * SH::P + 4 * iw));
        }
    }
    return prmt(prmt(p[0], p[1], 0x0073u), prmt(p[2], p[3], 0x0073u), 0x5410u);
}

template <class SH>
__device__ __forceinline__ uint32_t gather_word_rot(const uint32_t* __restrict__ S, uint32_t iw, uint32_t jw, uint32_t rot)
{
    if constexpr (SH::EB == 2) return gather_word<SH>(S, iw, jw);
    uint32_t word = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint32_t jj = ((uint32_t)j + rot) & 3u;
        word |= (row_bits_top(*reinterpret_cast<const uint4*>(S + (4 * jw + jj) * SH::P + 4 * iw)) >> 24) << (8u * jj);
    }
    return word;
}

// an (x | y << 8) pair with both fields below 256 in the register format of this shape
template <class SH>
__device__ __forceinline__ constexpr uint32_t widen(uint32_t f)
{
    return SH::WIDE ? ((f & 0xFFu) | ((f & 0xFF00u) << 8)) : f;
}

// entry index soff + y*P + x of the site packed as v = x | y << YSH (fields may hold x + D, y + D: cells wrap inside
// the domain, R14): mask both fields at once, then one byte dot product (x, y, 0, 0) . (1, P, 0, 0) + soff (D = 256: the
// pitch is no byte weight, shift and multiply-add)
template <class SH>
__device__ __forceinline__ uint32_t site_index(uint32_t v, uint32_t soff)
{
    const uint32_t vm = v & (uint32_t)((SH::D - 1) | ((SH::D - 1) << SH::YSH));
    if constexpr (SH::WIDE) {
        return (vm >> 16) * (uint32_t)SH::P + (vm & 0xFFFFu) + soff;
    } else {
        static_assert(SH::WIDE || SH::P <= 255, "the pitch is a byte weight of the dot product");
        return __dp4a(vm, (uint32_t)(1 | (SH::P << 8)), soff);
    }
}

// Carry out an accepted update at entry index `i` (relative to Sb): the site's four links flip.
// up = true: deposition (minimum -> maximum), false: removal.
template <class SH>
__device__ __forceinline__ void flip_links(uint32_t* Sb, uint32_t i, bool up)
{
    if constexpr (SH::EB == 2) {
        unsigned char* B2 = reinterpret_cast<unsigned char*>(Sb) + 2u * i;
        *reinterpret_cast<unsigned short*>(B2) = up ? 0xFFFF : 0;      // own W and S links
        B2[2] = up ? 0 : 0xFF;                                         // east neighbour's W link = sigma_x(x+1,y)
        B2[2 * SH::P + 1] = up ? 0 : 0xFF;                             // north neighbour's S link = sigma_y(x,y+1)
        return;
    }
    unsigned char* B = reinterpret_cast<unsigned char*>(Sb + i);
    const unsigned char v1 = up ? 0xFF : 0, v0 = up ? 0 : 0xFF;
    Sb[i] = up ? kEntryMax : kEntryMin;
    B[-4 + 1] = v1;                 // west neighbour's E link  = sigma_x(x,y)
    B[+4 + 0] = v0;                 // east neighbour's W link  = sigma_x(x+1,y)
    B[-4 * SH::P + 3] = v1;         // south neighbour's N link = sigma_y(x,y)
    B[+4 * SH::P + 2] = v0;         // north neighbour's S link = sigma_y(x,y+1)
}

// The same for a decision d in {-1, 0, +1} that differs from lane to lane in value AND direction (both rates non-zero):
// written as predicated stores by hand -- left to the compiler, the `if (d != 0)` around stores whose values depend on d
// becomes a divergent branch per cell and phase (BSSY / BRA / BSYNC; the mixed-rate sweep then ran 5x slower than p = 1).
template <class SH>
__device__ __forceinline__ void flip_links_signed(uint32_t* Sb, uint32_t i, int d)
{
    const bool up = d > 0;
    if constexpr (SH::EB == 2) {
        const uint32_t a = (uint32_t)__cvta_generic_to_shared(Sb) + 2u * i;
        const uint32_t e = up ? 0xFFFFu : 0u, v0 = up ? 0u : 0xFFu;
        asm volatile(
            "{\n\t.reg .pred p;\n\tsetp.ne.s32 p, %0, 0;\n\t"
            "@p st.shared.u16 [%1], %2;\n\t"          // own W and S links
            "@p st.shared.u8 [%1+2], %3;\n\t"         // east neighbour's W link
            "@p st.shared.u8 [%1+%4], %3;\n\t}"       // north neighbour's S link
            :: "r"(d), "r"(a), "r"(e), "r"(v0), "n"(2 * SH::P + 1) : "memory");
    } else {
        const uint32_t a = (uint32_t)__cvta_generic_to_shared(Sb + i);
        const uint32_t e = up ? kEntryMax : kEntryMin, v1 = up ? 0xFFu : 0u, v0 = up ? 0u : 0xFFu;
        asm volatile(
            "{\n\t.reg .pred p;\n\tsetp.ne.s32 p, %0, 0;\n\t"
            "@p st.shared.u32 [%1], %2;\n\t"
            "@p st.shared.u8 [%1+-3], %3;\n\t"        // west neighbour's E link
            "@p st.shared.u8 [%1+4], %4;\n\t"         // east neighbour's W link
            "@p st.shared.u8 [%1+%5], %3;\n\t"        // south neighbour's N link
            "@p st.shared.u8 [%1+%6], %4;\n\t}"       // north neighbour's S link
            :: "r"(d), "r"(a), "r"(e), "r"(v1), "r"(v0), "n"(-4 * SH::P + 3), "n"(4 * SH::P + 2) : "memory");
    }
}

// Acceptance rule of one launch.  ONEDIR: only one of p, q is non-zero (always so for the sync variant),
// so a single entry pattern is tested and the stored values are launch constants; ALWAYS: that live
// threshold is 65536 (p = 1 or q = 1) and the 16-bit comparison is dropped as well.
template <bool ONEDIR, bool ALWAYS, int EB = 4>
struct Rule {
    static constexpr uint32_t kMin = EB == 4 ? kEntryMin : kEntry2Min, kMax = EB == 4 ? kEntryMax : kEntry2Max;
    uint32_t P16, Q16, target, T16;
    bool dep;
    __device__ __forceinline__ Rule(uint32_t p16, uint32_t q16)
        : P16(p16), Q16(q16), target(q16 == 0u ? kMin : kMax), T16(q16 == 0u ? p16 : q16), dep(q16 == 0u) {}
    // decision for entry value e and attempt word w: 0 nothing, +1 deposit, -1 remove
    __device__ __forceinline__ int decide(uint32_t e, uint32_t w) const
    {
        if constexpr (ONEDIR) {
            bool acc = e == target;
            if constexpr (!ALWAYS) acc = acc && (w >> 16) < T16;
            return acc ? (dep ? 1 : -1) : 0;
        } else {
            const uint32_t r16 = w >> 16;                 // (no short-circuit operators: they compile to branches)
            return (int)((e == kMin) & (r16 < P16)) - (int)((e == kMax) & (r16 < Q16));
        }
    }
    // carry out decision d at entry i and count it in net (deposits - removals; ONEDIR counts updates, the caller signs them)
    template <class SH>
    __device__ __forceinline__ void apply(uint32_t* Sb, uint32_t i, int d, int& net) const
    {
        if constexpr (ONEDIR) { if (d != 0) { flip_links<SH>(Sb, i, dep); ++net; } }
        else { flip_links_signed<SH>(Sb, i, d); net += d; }
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

// The collective single-hit steps of one domain sweep (:168-174).
// DEAD: dead-border device layer (:135): attempts whose domain-local x or y is >= dead_lim are not carried out.
// S = row 0 of the window, soff = entry index of the domain's site (0,0) in it.  Returns deposits - removals of the
// calling lane's cells.
template <class SH, int BLK, bool ONEDIR, bool ALWAYS, bool DEAD>
__device__ __forceinline__ int run_steps(uint32_t* __restrict__ S, uint32_t soff, uint32_t* __restrict__ BT, uint32_t tg, int grp, uint32_t wmask,
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
        cellc[j] = ((c & (SH::NCX - 1)) * CX) | (((c >> LOG2NCX) * CY) << SH::YSH);
    }
    const Rule<ONEDIR, ALWAYS, SH::EB> rule(P16, Q16);

    // decision for the site packed in v (x | y << YSH before wrapping); idx receives its entry index.  `live` = this cell
    // takes part in the current phase (delayed borders): the loads are predicated, everything else is straight-line code, so
    // a phase is no divergent branch.  An entry value of 0x55555555 is neither a minimum nor a maximum.
    auto load_site = [&](uint32_t v, uint32_t& idx, bool live = true) -> uint32_t {
        idx = site_index<SH>(v, soff);
        if constexpr (DEAD) {
            const uint32_t vm = v & (uint32_t)((SH::D - 1) | ((SH::D - 1) << SH::YSH));
            live = live && (vm & (SH::WIDE ? 0xFFFFu : 0xFFu)) < dead_lim && (vm >> SH::YSH) < dead_lim;      // dead border: not carried out
        }
        uint32_t e = 0x55555555u;
        if constexpr (SH::EB == 2) {
            const unsigned char* B2 = reinterpret_cast<const unsigned char*>(S) + 2u * idx;
            if (live) e = (uint32_t)*reinterpret_cast<const unsigned short*>(B2) | ((uint32_t)B2[2] << 16) | ((uint32_t)B2[2 * SH::P + 1] << 24);   // (W, S, E, N)
        } else {
            if (live) e = S[idx];
        }
        return e;
    };
    auto decide_site = [&](uint32_t v, uint32_t w, uint32_t& idx, bool live = true) -> int { return rule.decide(load_site(v, idx, live), w); };
    int net = 0;                                     // accepted updates of this lane's cells (counted under the stores' predicate)

    // a few groups of four steps per loop trip: the next groups' Philox rounds fill the issue slots the current
    // group's shared-memory round trips leave open (+3 % at D = 64, +8 % at D = 128 over no unrolling)
#ifndef OCT_DELAYED_UNROLL
#define OCT_DELAYED_UNROLL 1
#endif
    // (delayed borders run three phases per step: one group of four steps per trip keeps the loop in the instruction cache)
    constexpr int kUnrollK4 = BLK == kBlkDelayed ? OCT_DELAYED_UNROLL : CPT >= 4 ? 2 : (SH::BTW / 4 < 8 / CPT ? SH::BTW / 4 : 8 / CPT);
    constexpr uint32_t RB = SH::BTW / 4;             // groups of four steps per fill of the block-step ring
#pragma unroll 1
    for (uint32_t kb = k4_begin; kb < k4_end; kb += RB) {
    // ---- a3: block-step words of the next BTW steps (:170, :172; R13/R17/R24); the previous step ended with a barrier
    for (uint32_t q = tg; q < RB && kb + q < k4_end; q += G) {
        uint32_t o[4];
        philox4x32_10(kb + q, 0u, c2b, t, rk, o);
        // what the steps need of a block-step word is worked out here, once per step instead of once per warp and step:
        // DB: the cell origin (ox, oy) (R13); DT: the quadrant's offset (R17), DTr: plus the origin (:234, R26)
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
            if constexpr (BLK == kBlkDT)
                o[kk] = widen<SH>(((((o[kk] >> 16) & 1u) * (CX / 2)) | ((((o[kk] >> 17) & 1u) * (CY / 2)) << 8))
                                  + (o[kk] & dtr_mask & (uint32_t)((CX - 1) | ((CY - 1) << 8))));
            else
                o[kk] = widen<SH>(o[kk] & FM);
        }
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
                const uint32_t sc = Bw;
                int dec[CPT];
#pragma unroll
                for (int j = 0; j < CPT; ++j) {
                    const uint32_t w = rw[j][kk];
                    dec[j] = decide_site(widen<SH>(w & FM) + cellc[j] + sc, w, idx[j]);
                }
                links_sync<G, SH::DPB>(grp, wmask);
#pragma unroll
                for (int j = 0; j < CPT; ++j) rule.template apply<SH>(S, idx[j], dec[j], net);
                links_sync<G, SH::DPB>(grp, wmask);
            } else if constexpr (BLK == kBlkDelayed) {
                // delayed borders (:174): bulk, then edges, then corners (R15)
                const uint32_t sc = Bw;
                uint32_t cls[CPT], vv[CPT];
#pragma unroll
                for (int j = 0; j < CPT; ++j) {
                    const uint32_t f = rw[j][kk] & FM;
                    vv[j] = widen<SH>(f) + cellc[j] + sc;
                    cls[j] = (uint32_t)((f & 0xFFu) == (uint32_t)(CX - 1)) + (uint32_t)((f >> 8) == (uint32_t)(CY - 1));
                }
                // The three phases only matter when two of the sites selected in this step are nearest neighbours (an update changes
                // the four links of its site and nothing else, and a decision reads only the four links of its site): without such
                // a pair every order gives the same lattice, and the step is ONE load-decide-store pass instead of three dependent
                // ones.  A selected site's east (north) neighbour can only have been selected by the cell east (north) of it, so
                // where a domain's cells sit in one warp two shuffles per cell slot find every pair; ~4 of 5 steps have none.
                // The entries of all cells are loaded first (they are what the bulk phase, or the single pass, decides on), the
                // shuffles run under the loads' latency.
                uint32_t ent[CPT];
#pragma unroll
                for (int j = 0; j < CPT; ++j) ent[j] = load_site(vv[j], idx[j]);
                bool phased = true;
                if constexpr (G <= 32 && SH::NCX <= G && !SH::WIDE) {
                    constexpr uint32_t WRAP = (uint32_t)((SH::D - 1) | ((SH::D - 1) << 8));
                    const uint32_t lane_base = (threadIdx.x & 31u) & ~(uint32_t)(G - 1);      // G = 16: the half warp of this domain
                    bool pair = false;
#pragma unroll
                    for (int j = 0; j < CPT; ++j) {
                        const uint32_t c = tg + j * G;
                        const uint32_t ce = (c & ~(uint32_t)(SH::NCX - 1)) | ((c + 1u) & (uint32_t)(SH::NCX - 1));   // cell east of c (same slot)
                        const uint32_t cn = (c + SH::NCX) & (uint32_t)(SH::NCELL - 1);                              // cell north of c
                        const uint32_t me = vv[j] & WRAP;
                        const uint32_t east = __shfl_sync(wmask, vv[j], lane_base | (ce & (uint32_t)(G - 1))) & WRAP;
                        uint32_t north = 0u;
#pragma unroll
                        for (int jj = 0; jj < CPT; ++jj) {
                            const uint32_t got = __shfl_sync(wmask, vv[jj], lane_base | (cn & (uint32_t)(G - 1)));
                            if ((int)(cn / G) == jj) north = got & WRAP;
                        }
                        // (x = D - 1 or y = D - 1: me + 1 / me + 256 leaves the field, no wrapped coordinate equals it -- the halo is inactive)
                        pair = pair || east == me + 1u || north == me + 256u;
                    }
                    phased = __any_sync(wmask, pair);
                }
                {
                    // bulk phase, or (no nearest-neighbour pair) every cell: decisions on the entries loaded above
                    int dec[CPT];
#pragma unroll
                    for (int j = 0; j < CPT; ++j) dec[j] = rule.decide((phased && cls[j] != 0u) ? 0x55555555u : ent[j], rw[j][kk]);
#pragma unroll
                    for (int j = 0; j < CPT; ++j) rule.template apply<SH>(S, idx[j], dec[j], net);
                    links_sync<G, SH::DPB>(grp, wmask);
                }
                if (phased) {
#pragma unroll
                    for (uint32_t phase = 1; phase < 3; ++phase) {
                        int dec[CPT];                    // cells of one phase never touch common links (R15): loads first
#pragma unroll
                        for (int j = 0; j < CPT; ++j) dec[j] = decide_site(vv[j], rw[j][kk], idx[j], cls[j] == phase);
#pragma unroll
                        for (int j = 0; j < CPT; ++j) rule.template apply<SH>(S, idx[j], dec[j], net);
                        links_sync<G, SH::DPB>(grp, wmask);
                    }
                }
            } else {
                // block-layer DT (:170): one random quadrant of every cell per step (R17).  The cells of a step
                // cannot interact, so all loads go first and the stores follow (no load waits behind a store)
                // (block-layer DTr, :234 / R26: plus the per-step origin of block-layer DB; site_index wraps, R14)
                const uint32_t qc = Bw;
                int dec[CPT];
#pragma unroll
                for (int j = 0; j < CPT; ++j) {
                    const uint32_t w = rw[j][kk];
                    dec[j] = decide_site(widen<SH>(w & FM) + cellc[j] + qc, w, idx[j]);
                }
#pragma unroll
                for (int j = 0; j < CPT; ++j) rule.template apply<SH>(S, idx[j], dec[j], net);
                links_sync<G, SH::DPB>(grp, wmask);
            }
        }
    }
    }
    return ONEDIR && !rule.dep ? -net : net;
}

// number of set W links of the sites (0..n00-1, y00) of the domain: with n00 = x00 + 1 it is h(x00,y00) minus the
// height of the inactive site west of the row start, up to a constant (used before and after the sweep, R20)
template <class SH>
__device__ __forceinline__ int row_links_up(const uint32_t* Sb, uint32_t n00, uint32_t y00, uint32_t tg)
{
    int n = 0;
    if constexpr (SH::EB == 2) {       // Sb = entry (0,0) of the domain as a two-byte entry pointer
        const unsigned char* B = reinterpret_cast<const unsigned char*>(Sb);
        for (uint32_t x = tg; x < n00; x += SH::G) n += (int)(B[2u * (y00 * SH::P + x)] & 1u);
    } else {
        for (uint32_t x = tg; x < n00; x += SH::G) n += (int)(Sb[y00 * SH::P + x] & 1u);
    }
    return n;
}

__device__ __forceinline__ const SweepParams& common_params(const SweepParams& p) { return p; }
__device__ __forceinline__ const SweepParams& common_params(const SweepBatchParams& p) { return p.common; }

// DEAD = false: tiled device layers DTr / DT (four launches per MCS, one per domain set);
// DEAD = true : dead-border device layers DB / cDB / DBh (all tiles in one launch; the rim of width dead_w is
//               never updated, and words shared with the next tile are neither read, counted nor written, :166).
template <int LOG2D, int TCX, int TCY, int BLK, int G_, int DPB, bool DEAD, bool BATCH = false, int EB = 4>
__global__ void __launch_bounds__(LinkShape<LOG2D, TCX, TCY, G_, DPB, EB>::NTHREADS)
sweep_links_kernel(const __grid_constant__ typename std::conditional<BATCH, SweepBatchParams, SweepParams>::type PP)
{
    using SH = LinkShape<LOG2D, TCX, TCY, G_, DPB, EB>;
    constexpr int D = SH::D, G = SH::G, NW = SH::NW;

    extern __shared__ __align__(16) uint32_t smem_raw[];
    const int grp = threadIdx.x / G;                 // worker group inside the CTA
    const uint32_t tg = threadIdx.x % G;             // thread inside the group
    uint32_t* S0 = smem_raw + grp * (SH::SMEM_PER_DOMAIN / 4);
    uint32_t* S = EB == 4 ? S0 + SH::P : S0;         // row 0 of the window (four-byte entries: one spare row below it)
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
    // entry of the domain's site (0,0) (two-byte entries: half as many words in)
    uint32_t* Sb = EB == 4 ? S + offy * SH::P + offx : reinterpret_cast<uint32_t*>(reinterpret_cast<unsigned short*>(S) + offy * SH::P + offx);
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
            uint32_t e1 = 0u, e2 = 0u;                 // (two-byte entries hold no neighbour links: nothing to fetch)
            if constexpr (EB == 4) {
                e1 = __shfl_down_sync(wmask, A[jw], 1, 16);
                e2 = jw < 16 ? __shfl_sync(wmask, C, jw, 16) : __shfl_sync(wmask, C16, 0, 16);
            }
            expand_word<SH>(S, iw, jw, A[jw], iw == 15u ? e2 : e1, A[jw + 1]);
        }
        // last column: lane jw expands word (16, jw), lane 0 then (16, 16); its north word is the next lane's
        uint32_t Cn = 0u, Cn15 = 0u;
        if constexpr (EB == 4) { Cn = __shfl_down_sync(wmask, C, 1, 16); Cn15 = __shfl_sync(wmask, C16, 0, 16); }
        expand_word_rot<SH>(S, NW - 1, tg, C, 0u, tg == 15u ? Cn15 : Cn, tg >> 1);
        if (tg == 0u) {
            expand_word<SH>(S, NW - 1, NW - 1, C16, 0u, 0u);
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
            uint32_t e1 = 0u, e2 = 0u, Nw = 0u;
            if constexpr (EB == 4) {
                e1 = __shfl_down_sync(0xFFFFFFFFu, A[it], 1); e2 = __shfl_sync(0xFFFFFFFFu, C, jw);
                Nw = __shfl_xor_sync(0xFFFFFFFFu, hi ? A[it] : A[it + 1], 16);
            }
            if (jw < (uint32_t)NW) {
                expand_word<SH>(S, iw, jw, A[it], iw == 15u ? e2 : e1, Nw);
            }
        }
        uint32_t Cn = 0u;
        if constexpr (EB == 4) Cn = __shfl_down_sync(0xFFFFFFFFu, C, 1);
        if (tg < (uint32_t)NW) {
            expand_word_rot<SH>(S, NW - 1, tg, C, 0u, Cn, tg >> 1);       // the east links of this column are never read
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
                    if constexpr (EB == 2) {          // two-byte entries: own links only
                        if (kept(iw, jw)) A[it] = *word_ptr(iw, jw);
                    } else if constexpr (DEAD) {
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
    const uint32_t soff = offy * SH::P + offx;      // entry index of the domain's site (0,0)
    int net = 0;                                     // deposits - removals of this lane's cells
#define OCT_RUN(ONEDIR, ALWAYS) \
    run_steps<SH, BLK, ONEDIR, ALWAYS, DEAD>(S, soff, BT, tg, grp, wmask, c2b, c2c, t, rk, P.P16, P.Q16, P.dtr_mask, dead_lim, k4_begin, k4_end)
    if (onedir && T16 == 65536u) net = OCT_RUN(true, true);
    else if (onedir)             net = OCT_RUN(true, false);
    else if constexpr (BLK != kBlkSync) net = OCT_RUN(false, false);
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
        }
        if (kept(NW - 1, tg)) {
            const uint32_t word = gather_word_rot<SH>(S, NW - 1, tg, tg >> 1);
            put_word(NW - 1, tg, word);
        }
        if (tg == 0u && kept(NW - 1, NW - 1)) {
            const uint32_t word = gather_word<SH>(S, NW - 1, NW - 1);
            put_word(NW - 1, NW - 1, word);
        }
    } else if constexpr (SH::FAST_17) {
        const uint32_t hi = tg >> 4, iw = tg & 15u;
#pragma unroll 3
        for (uint32_t jw = hi; jw < (uint32_t)NW; jw += 2) {
            if (!kept(iw, jw)) continue;
            const uint32_t word = gather_word<SH>(S, iw, jw);
            put_word(iw, jw, word);
        }
        if (tg < (uint32_t)NW && kept(NW - 1, tg)) {
            const uint32_t word = gather_word_rot<SH>(S, NW - 1, tg, tg >> 1);
            put_word(NW - 1, tg, word);
        }
    } else {
        for (uint32_t idx = tg; idx < (uint32_t)(NW * NW); idx += G) {
            const uint32_t jw = idx / NW, iw = idx - jw * NW;
            if (!kept(iw, jw)) continue;
            const uint32_t word = gather_word<SH>(S, iw, jw);
            put_word(iw, jw, word);
        }
    }

    // counters: net deposits (counted by run_steps, one atomic per warp) and the tracked height of site (0,0): the site west
    // of the row start is inactive in this launch, so the change of h(0,0) is twice the change of the
    // number of up-links between them
    d00 += row_links_up<SH>(Sb, n00, r00, tg);
    if (d00 != 0) atomicAdd(&counters[1], (unsigned long long)(long long)(2 * d00));
    net = __reduce_add_sync(wmask, net);
    if ((threadIdx.x & 31) == 0 && net != 0) atomicAdd(&counters[0], (unsigned long long)(long long)net);
}

}  // namespace octb

// liboct_b200: host side of the C ABI declared in include/oct.h.  Argument checking, launch
// configuration and stream plumbing only -- every step of the hot path runs in the kernels of
// sweep.cuh and observe.cuh.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>

#include <cuda_runtime.h>

#include "../../include/oct.h"
#include "observe.cuh"
#include "observe_rows.cuh"
#include "philox.cuh"
#include "launch.h"
#include "sweep.cuh"

using namespace octb;

constexpr size_t kWsHeader = 256 + 2 * kColMaxBlocks * sizeof(int32_t);

struct oct_ctx {
    uint32_t L = 0, log2L = 0;
    uint64_t seed = 0;
    uint64_t t = 0;
    uint32_t* lat = nullptr;
    unsigned char* ws = nullptr;
    uint64_t launches = 0;
    int opt_kernel = OCT_KERNEL_AUTO;
    PhiloxRoundKeys rk{};
    std::string last_error;
    // oct_sweep_batch: helper stream and fork / join events, created on first use (handle 0 of the batch owns them)
    cudaStream_t aux = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;

    unsigned long long* counters() const { return reinterpret_cast<unsigned long long*>(ws); }
    // workspace: [0, 16) counters; [256, 1280) net slope of every CTA's part of column 0 (two lattices); then the arrays
    int32_t* blocksum() const { return reinterpret_cast<int32_t*>(ws + 256); }
    int32_t* anchorA() const { return reinterpret_cast<int32_t*>(ws + kWsHeader); }
    int32_t* anchorB() const { return reinterpret_cast<int32_t*>(ws + kWsHeader + (size_t)L * 4); }
    uint32_t* colA() const { return reinterpret_cast<uint32_t*>(ws + kWsHeader + (size_t)L * 8); }    // column 0, gathered (L/4 words)
    uint32_t* colB() const { return reinterpret_cast<uint32_t*>(ws + kWsHeader + (size_t)L * 9); }
};

namespace {

constexpr uint32_t kMinL = 16, kMaxL = 1u << 17;

bool valid_L(uint32_t L) { return L >= kMinL && L <= kMaxL && (L & (L - 1)) == 0; }

uint32_t ilog2(uint32_t v) { uint32_t r = 0; while ((1u << r) < v) ++r; return r; }

// probability -> 16-bit acceptance threshold, accept iff r16 < P16 (R18)
uint32_t prob16(double p)
{
    const double v = p * 65536.0 + 0.5;
    return v >= 65536.0 ? 65536u : static_cast<uint32_t>(v);
}

int fail_cuda(oct_ctx* c, cudaError_t e, const char* what)
{
    if (c) c->last_error = std::string(what) + ": " + cudaGetErrorString(e);
    return OCT_ECUDA;
}

#define OCT_CUDA(ctx, call)                                         \
    do {                                                            \
        cudaError_t e__ = (call);                                   \
        if (e__ != cudaSuccess) return fail_cuda(ctx, e__, #call);  \
    } while (0)

// ---- sweep kernel dispatch (the kernels are instantiated in sweep_inst.cu, one object per family and size) ----
bool find_launch(int ld, int tx, int ty, int blk, SweepLaunch* out)
{
    switch (ld) {
        case 5: return oct_find_packed_5(tx, ty, blk, out);
        case 6: return oct_find_packed_6(tx, ty, blk, out);
        case 7: return oct_find_packed_7(tx, ty, blk, out);
        case 8: return oct_find_packed_8(tx, ty, blk, out);
        default: return false;
    }
}

bool find_links_launch(int ld, int tx, int ty, int blk, bool variant_b, bool dead, SweepLaunch* out)
{
    switch (ld) {
        case 5: return oct_find_links_5(tx, ty, blk, variant_b, dead, out);
        case 6: return oct_find_links_6(tx, ty, blk, variant_b, dead, out);
        case 7: return oct_find_links_7(tx, ty, blk, variant_b, dead, out);
        case 8: return oct_find_links_8(tx, ty, blk, variant_b, dead, out);
        default: return false;
    }
}

struct SchemeFields {
    uint32_t dev, blk, tcx, tcy, log2D, ka, w;
    // dead-border layers: intervals per sweep as a power of two (DBh = DB with two) and the border width in sites
    uint32_t ka_eff() const { return dev == OCT_DEV_DBH ? 1u : ka; }
    uint32_t width() const { return w ? w : (dev == OCT_DEV_CDB ? 1u : 5u); }
};

SchemeFields split_scheme(int scheme)
{
    const uint32_t s = static_cast<uint32_t>(scheme);
    return {s & 15u, (s >> 4) & 15u, (s >> 8) & 15u, (s >> 12) & 15u, (s >> 16) & 31u, (s >> 21) & 3u, (s >> 23) & 7u};
}

int check_scheme(uint32_t L, int scheme)
{
    if (scheme < 0 || !valid_L(L)) return OCT_EINVAL;
    const SchemeFields f = split_scheme(scheme);
    if ((static_cast<uint32_t>(scheme) >> 26) != 0) return OCT_EINVAL;
    if (f.dev > 4 || f.blk > 3) return OCT_EINVAL;
    if (f.log2D < 5 || f.log2D > 8) return OCT_EINVAL;
    const uint32_t D = 1u << f.log2D, cx = 4u << f.tcx, cy = 4u << f.tcy;
    // t_async and border width belong to DB / cDB (DBh is DB with ka = 1); at most four intervals (they share the 2-bit
    // set field of the counters, R19), each made of whole Philox calls (4 steps)
    if ((f.ka || f.w) && f.dev != OCT_DEV_DB && f.dev != OCT_DEV_CDB) return OCT_EINVAL;
    if (f.ka > 2 || f.w >= D || ((cx * cy) >> f.ka) < 4 || ((cx * cy) >> f.ka) % 4 != 0) return OCT_EINVAL;
    if (cx > D || cy > D || cx > 64 || cy > 64) return OCT_EINVAL;
    const bool blk_dt = f.blk == OCT_BLK_DT || f.blk == OCT_BLK_DTR;
    if (blk_dt && (f.tcx < 1 || f.tcy < 1)) return OCT_EINVAL;   // :182
    // DT / DTr tile the lattice with 2D x 2D tiles; the dead-border layers with D x D tiles (a single tile, L = D, is
    // allowed: its window wraps onto itself only in the dead rim, which is neither tested nor written back)
    if (f.dev <= OCT_DEV_DT ? L < 2 * D : L < D) return OCT_EINVAL;
    SweepLaunch sl;
    if (!find_launch((int)f.log2D, (int)f.tcx, (int)f.tcy, blk_dt ? kBlkDT : kBlkSync, &sl)) return OCT_EINVAL;
    return OCT_OK;
}

int ensure_device(oct_ctx* c)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda(c, e, "cudaGetDevice");
    int major = 0;
    e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) return fail_cuda(c, e, "cudaDeviceGetAttribute");
    if (major != 10) {
        if (c) c->last_error = "device is not compute capability 10.x (sm_100a build)";
        return OCT_ECUDA;
    }
    return OCT_OK;
}

// one warp per word-row; 16 words per lane per chunk once a row holds at least one full chunk
template <int WHAT>
void launch_rows_what(const RowsParams& rp, uint32_t LW, cudaStream_t st)
{
    const unsigned blocks = (LW + kRows2Warps - 1) / kRows2Warps;
    if (LW >= 512u) rows3_kernel<WHAT, 16><<<blocks, kRows2Warps * 32, 0, st>>>(rp);
    else            rows3_kernel<WHAT, 4><<<blocks, kRows2Warps * 32, 0, st>>>(rp);
}

template <int WHAT>
void launch_rows_batch_what(const ObsBatchParams& bp, uint32_t nb, uint32_t LW, cudaStream_t st)
{
    const dim3 grid((LW + kRows2Warps - 1) / kRows2Warps, nb);
    if (LW >= 512u) rows3_batch_kernel<WHAT, 16><<<grid, kRows2Warps * 32, 0, st>>>(bp);
    else            rows3_batch_kernel<WHAT, 4><<<grid, kRows2Warps * 32, 0, st>>>(bp);
}

void launch_rows_batch(int what, const ObsBatchParams& bp, uint32_t nb, uint32_t LW, cudaStream_t st)
{
    switch (what) {
        case 1: launch_rows_batch_what<1>(bp, nb, LW, st); break;
        case 2: launch_rows_batch_what<2>(bp, nb, LW, st); break;
        case 3: launch_rows_batch_what<3>(bp, nb, LW, st); break;
        case 4: launch_rows_batch_what<4>(bp, nb, LW, st); break;
        case 5: launch_rows_batch_what<5>(bp, nb, LW, st); break;
        case 6: launch_rows_batch_what<6>(bp, nb, LW, st); break;
        case 7: launch_rows_batch_what<7>(bp, nb, LW, st); break;
        default: break;
    }
}

void launch_rows(int what, const RowsParams& rp, uint32_t LW, cudaStream_t st)
{
    switch (what) {
        case 1: launch_rows_what<1>(rp, LW, st); break;
        case 2: launch_rows_what<2>(rp, LW, st); break;
        case 3: launch_rows_what<3>(rp, LW, st); break;
        case 4: launch_rows_what<4>(rp, LW, st); break;
        case 5: launch_rows_what<5>(rp, LW, st); break;
        case 6: launch_rows_what<6>(rp, LW, st); break;
        case 7: launch_rows_what<7>(rp, LW, st); break;
        default: break;
    }
}

// column anchors of the current lattice (and of a snapshot, latB != nullptr) into the handle's workspace: 2 small launches;
// the second one also zeroes the n_zero int64 words at `zero` (the output of the reduction that follows)
int launch_anchors(oct_ctx* c, const uint32_t* latB, cudaStream_t st, void* zero = nullptr, int n_zero = 0)
{
    const uint32_t LW = c->L >> 2, nlat = latB ? 2u : 1u;
    const dim3 grid((LW + kColThreads - 1) / kColThreads, nlat);
    column_gather_kernel<<<grid, kColThreads, 0, st>>>(c->lat, latB, c->L, c->colA(), c->colB(), c->blocksum());
    column_anchor_kernel<<<grid, kColThreads, 0, st>>>(c->colA(), c->colB(), c->blocksum(), c->L, c->anchorA(), c->anchorB(),
                                                      static_cast<unsigned long long*>(zero), n_zero);
    c->launches += 2;
    OCT_CUDA(c, cudaGetLastError());
    return OCT_OK;
}

}  // namespace

extern "C" {

size_t oct_lattice_bytes(uint32_t L) { return valid_L(L) ? (size_t)L * L / 4 : 0; }

size_t oct_workspace_bytes(uint32_t L) { return valid_L(L) ? kWsHeader + 10 * (size_t)L : 0; }   // header; 2 x L int32 anchors; 2 x L/4 words of column 0

int oct_create(oct_ctx** out, uint32_t L, uint64_t seed, int init, void* lattice_dev, void* workspace_dev, void* stream)
{
    if (!out) return OCT_EINVAL;
    *out = nullptr;
    if (!valid_L(L) || !lattice_dev || !workspace_dev) return OCT_EINVAL;
    if (init != OCT_INIT_FLAT && init != OCT_INIT_FLAT_SHIFTED && init != OCT_INIT_FROM_DEVICE) return OCT_EINVAL;
    if ((reinterpret_cast<uintptr_t>(lattice_dev) & 15u) || (reinterpret_cast<uintptr_t>(workspace_dev) & 15u)) return OCT_EINVAL;
    oct_ctx* c = new (std::nothrow) oct_ctx;
    if (!c) return OCT_ENOMEM;
    c->L = L; c->log2L = ilog2(L); c->seed = seed; c->t = 0;
    c->lat = static_cast<uint32_t*>(lattice_dev);
    c->ws = static_cast<unsigned char*>(workspace_dev);
    c->rk = make_round_keys(seed);
    int rc = ensure_device(c);
    if (rc != OCT_OK) { delete c; return rc; }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    cudaError_t e = cudaMemsetAsync(c->ws, 0, 256, st);
    if (e == cudaSuccess && init != OCT_INIT_FROM_DEVICE) {
        const size_t n_vec = (size_t)L * L / 4 / 16;
        const unsigned blocks = (unsigned)((n_vec + 255) / 256 < 148 * 8 ? (n_vec + 255) / 256 : 148 * 8);
        fill_words_kernel<<<blocks, 256, 0, st>>>(reinterpret_cast<uint4*>(c->lat), n_vec,
                                                  init == OCT_INIT_FLAT ? 0x33CC33CCu : 0xCC33CC33u);
        c->launches++;
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) { delete c; return OCT_ECUDA; }
    *out = c;
    return OCT_OK;
}

int oct_set_state(oct_ctx* c, uint64_t t_mcs, int64_t h00, int64_t net, void* stream)
{
    if (!c || t_mcs > 0xFFFFFFFFull) return OCT_EINVAL;
    set_counters_kernel<<<1, 1, 0, static_cast<cudaStream_t>(stream)>>>(c->counters(), h00, net);
    c->launches++;
    OCT_CUDA(c, cudaGetLastError());
    c->t = t_mcs;
    return OCT_OK;
}

int oct_scheme_supported(uint32_t L, int scheme) { return check_scheme(L, scheme); }

int oct_set_option(oct_ctx* c, int option, int value)
{
    if (!c) return OCT_EINVAL;
    if (option == OCT_OPT_KERNEL && value >= OCT_KERNEL_AUTO && value <= OCT_KERNEL_LINKS_B) { c->opt_kernel = value; return OCT_OK; }
    return OCT_EINVAL;
}

}  // extern "C"

namespace {

// Everything about a sweep call that does not depend on the lattice it runs on.
struct SweepPlan {
    SchemeFields f;
    SweepLaunch sl;
    uint32_t P16, Q16, ndom, grid, n_launch;
    bool pdl;                        // link-entry kernels wait for their predecessor themselves (griddepcontrol.wait)
};

int plan_sweep(oct_ctx* c, double p, double q, int scheme, SweepPlan* pl)
{
    if (!(p >= 0.0 && p <= 1.0) || !(q >= 0.0 && q <= 1.0)) return OCT_EINVAL;
    if (check_scheme(c->L, scheme) != OCT_OK) return OCT_EINVAL;
    pl->f = split_scheme(scheme);
    const SchemeFields& f = pl->f;
    pl->P16 = prob16(p); pl->Q16 = prob16(q);
    const int blk = (f.blk == OCT_BLK_DT || f.blk == OCT_BLK_DTR) ? kBlkDT
                  : (f.blk == OCT_BLK_DB_DELAYED || (pl->P16 > 0 && pl->Q16 > 0)) ? kBlkDelayed : kBlkSync;   // R16
    // the link-entry kernel serves every (D, TC) it is instantiated for (sweep_inst.cu: every shape the library accepts
    // except D = 32 TC=2,2, D = 256 as two-byte entries); the bit-packed kernel serves the rest and kernel option 1
    // one measured exception (profiles/r3_shapes.md): delayed borders at D = 256 with 128 cells per domain (TC=3,2 / 4,1) run
    // 11 % faster on the bit-packed kernel (one 128-thread CTA per SM cannot hide three CTA barriers per step)
    const bool packed_wins = f.log2D == 8 && f.tcx + f.tcy >= 5 && blk == kBlkDelayed && c->opt_kernel == OCT_KERNEL_AUTO;
    const bool links = c->opt_kernel != OCT_KERNEL_BITPACKED && !packed_wins &&
                       find_links_launch((int)f.log2D, (int)f.tcx, (int)f.tcy, blk, c->opt_kernel == OCT_KERNEL_LINKS_B,
                                         f.dev > OCT_DEV_DT, &pl->sl);
    if (!links && !find_launch((int)f.log2D, (int)f.tcx, (int)f.tcy, blk, &pl->sl)) return OCT_EINVAL;
    pl->pdl = links;
    const bool tiled = f.dev <= OCT_DEV_DT;
    const uint32_t nt = tiled ? c->L >> (f.log2D + 1) : c->L >> f.log2D;
    pl->ndom = nt * nt;
    pl->grid = (pl->ndom + pl->sl.dpb - 1) / pl->sl.dpb;
    pl->n_launch = tiled ? 4u : (1u << f.ka_eff());   // :144 one launch per domain set; dead borders: one per interval (R27)
    return OCT_OK;
}

// Kernels that need more than 48 KiB of dynamic shared memory must be opted in.  The attribute belongs to the function ON
// THE CURRENT DEVICE, so a process that drives several GPUs has to set it on each of them; remembering "done" per function
// pointer (as this code once did) leaves the second device without it and every large launch there fails.  Setting it
// costs a few microseconds next to the 4 * n_mcs launches of the call, so it is simply set on every sweep call: no cache,
// nothing shared between host threads.
int opt_in_smem(oct_ctx* c, const void* fn, int smem)
{
    if (smem <= 48 * 1024) return OCT_OK;
    OCT_CUDA(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    return OCT_OK;
}

// Launch a sweep kernel with programmatic stream serialisation: the kernel may be scheduled while its predecessor in
// the stream drains; it waits for the predecessor's completion (griddepcontrol.wait) before its first global access.
template <class PARAMS>
cudaError_t launch_sweep(void (*kern)(const PARAMS), dim3 grid, int threads, int smem, cudaStream_t st, const PARAMS& p, bool pdl)
{
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid; cfg.blockDim = dim3((unsigned)threads); cfg.dynamicSmemBytes = (size_t)smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1u : 0u;
    return cudaLaunchKernelEx(&cfg, kern, p);
}

void fill_common(SweepParams& sp, const oct_ctx* c, const SweepPlan& pl)
{
    sp.L = c->L; sp.log2L = c->log2L; sp.P16 = pl.P16; sp.Q16 = pl.Q16; sp.dev = pl.f.dev; sp.ndom = pl.ndom;
    sp.dtr_mask = pl.f.blk == OCT_BLK_DTR ? ~0u : 0u;
    sp.dead_w = pl.f.width(); sp.ka = pl.f.ka_eff();
}

}  // namespace

extern "C" {

int oct_sweep(oct_ctx* c, uint64_t n_mcs, double p, double q, int scheme, void* stream)
{
    if (!c) return OCT_EINVAL;
    SweepPlan pl;
    int rc = plan_sweep(c, p, q, scheme, &pl);
    if (rc) return rc;
    if (c->t + n_mcs > 0xFFFFFFFFull || c->t + n_mcs < c->t) return OCT_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    rc = opt_in_smem(c, reinterpret_cast<const void*>(pl.sl.kern), pl.sl.smem);
    if (rc) return rc;

    SweepParams sp{};
    fill_common(sp, c, pl);
    sp.lat = c->lat; sp.counters = c->counters(); sp.rk = c->rk;
    for (uint64_t i = 0; i < n_mcs; ++i) {
        sp.t = static_cast<uint32_t>(c->t);
        for (uint32_t si = 0; si < pl.n_launch; ++si) {   // :144 sync = kernel boundary after each set
            sp.si = si;
            OCT_CUDA(c, launch_sweep(pl.sl.kern, dim3(pl.grid), pl.sl.threads, pl.sl.smem, st, sp, pl.pdl));
            c->launches++;
        }
        OCT_CUDA(c, cudaGetLastError());   // on failure the clock stays at the sweeps completed so far (oct_mcs)
        c->t++;
    }
    return OCT_OK;
}

int oct_sweep_batch(oct_ctx* const* cs, uint32_t n, uint64_t n_mcs, double p, double q, int scheme, void* stream)
{
    if (!cs || n == 0) return OCT_EINVAL;
    for (uint32_t i = 0; i < n; ++i) {
        if (!cs[i] || cs[i]->L != cs[0]->L) return OCT_EINVAL;
        if (cs[i]->t + n_mcs > 0xFFFFFFFFull || cs[i]->t + n_mcs < cs[i]->t) return OCT_EINVAL;
        for (uint32_t j = 0; j < i; ++j) if (cs[j] == cs[i] || cs[j]->lat == cs[i]->lat) return OCT_EINVAL;
    }
    oct_ctx* c0 = cs[0];
    SweepPlan pl;
    int rc = plan_sweep(c0, p, q, scheme, &pl);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (!pl.sl.kern_batch) {
        // no many-lattices kernel for this shape: the members run one after the other (same results)
        for (uint32_t i = 0; i < n; ++i) {
            const int keep = cs[i]->opt_kernel;
            cs[i]->opt_kernel = c0->opt_kernel;
            rc = oct_sweep(cs[i], n_mcs, p, q, scheme, stream);
            cs[i]->opt_kernel = keep;
            if (rc) return rc;
        }
        return OCT_OK;
    }
    rc = opt_in_smem(c0, reinterpret_cast<const void*>(pl.sl.kern_batch), pl.sl.smem);
    if (rc) return rc;
    // Two halves of the ensemble run side by side, one on the caller's stream and one on a helper stream that forks from
    // it and joins it again below.  The launches of one half follow each other (kernel boundary = the synchronisation of
    // :144), and a launch of w waves of domains lasts ceil(w) domain-sweep times; the other half's launches fill that tail
    // (32 x L = 1024: 4.2e11 -> 5.0e11 attempts/s; 64 members and more run at the single-lattice rate).
    const uint32_t n_half = n >= 2 ? (n + 1) / 2 : n;
    const bool two = n >= 2;
    if (two && !c0->aux) {
        // all three or none: a handle with a helper stream but no events would fail on every later batch call
        cudaStream_t aux = nullptr;
        cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
        cudaError_t e = cudaStreamCreateWithFlags(&aux, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ev_fork, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ev_join, cudaEventDisableTiming);
        if (e != cudaSuccess) {
            if (ev_join) cudaEventDestroy(ev_join);
            if (ev_fork) cudaEventDestroy(ev_fork);
            if (aux) cudaStreamDestroy(aux);
            return fail_cuda(c0, e, "oct_sweep_batch: helper stream / events");
        }
        c0->aux = aux; c0->ev_fork = ev_fork; c0->ev_join = ev_join;
    }
    if (two) {
        OCT_CUDA(c0, cudaEventRecord(c0->ev_fork, st));
        OCT_CUDA(c0, cudaStreamWaitEvent(c0->aux, c0->ev_fork, 0));
    }
    SweepBatchParams bp{};
    fill_common(bp.common, c0, pl);
    cudaError_t e_launch = cudaSuccess;      // the first failure, kept: cudaGetLastError() hands an error out only once
    bool partial = false;                    // a failure after part of an MCS was enqueued
    for (uint64_t i = 0; i < n_mcs && e_launch == cudaSuccess; ++i) {
        uint32_t enq = 0;
        for (uint32_t half = 0; half < (two ? 2u : 1u) && e_launch == cudaSuccess; ++half) {
            const uint32_t h0 = half ? n_half : 0u, h1 = half ? n : n_half;
            cudaStream_t hs = half ? c0->aux : st;
            for (uint32_t m0 = h0; m0 < h1; m0 += kMaxBatch) {       // at most kMaxBatch members per launch
                const uint32_t nb = h1 - m0 < (uint32_t)kMaxBatch ? h1 - m0 : (uint32_t)kMaxBatch;
                for (uint32_t m = 0; m < nb; ++m) {
                    const oct_ctx* c = cs[m0 + m];
                    bp.m[m] = BatchMember{c->lat, c->counters(), (uint32_t)c->seed, (uint32_t)(c->seed >> 32), (uint32_t)c->t, 0u};
                }
                for (uint32_t si = 0; si < pl.n_launch && e_launch == cudaSuccess; ++si) {
                    bp.common.si = si;
                    e_launch = launch_sweep(pl.sl.kern_batch, dim3(pl.grid, nb), pl.sl.threads, pl.sl.smem, hs, bp, pl.pdl);
                    if (e_launch == cudaSuccess) { c0->launches++; ++enq; }
                }
            }
        }
        if (e_launch == cudaSuccess) e_launch = cudaGetLastError();
        if (e_launch == cudaSuccess)
            for (uint32_t m = 0; m < n; ++m) cs[m]->t++;
        else if (enq) partial = true;
    }
    if (two) {                                                       // join, whatever happened: the caller's stream stays the only one to wait on
        cudaEventRecord(c0->ev_join, c0->aux);
        cudaStreamWaitEvent(st, c0->ev_join, 0);
    }
    if (e_launch != cudaSuccess) {
        (void)cudaGetLastError();                                    // leave no stale error for the caller's next CUDA call
        // Some members may have received 1..3 of the 4 domain sets of the failing MCS while no clock was advanced for it:
        // their lattices are no longer a function of (seed, t).  Say so instead of pretending the state is resumable.
        const int rc_fail = fail_cuda(c0, e_launch, partial ? "oct_sweep_batch launch (members hold a partly enqueued MCS: re-create or re-upload them)"
                                                            : "oct_sweep_batch launch");
        return partial ? OCT_ESTATE : rc_fail;
    }
    return OCT_OK;
}

int oct_heights(oct_ctx* c, int32_t* heights_dev, void* stream)
{
    if (!c || !heights_dev || (reinterpret_cast<uintptr_t>(heights_dev) & 15u)) return OCT_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int rc = launch_anchors(c, nullptr, st);
    if (rc) return rc;
    RowsParams rp{};
    rp.latA = c->lat; rp.anchorA = c->anchorA(); rp.countersA = c->counters(); rp.heights = heights_dev; rp.L = c->L;
    const uint32_t LW = c->L >> 2;
    heights_kernel<4><<<(LW + kRows2Warps - 1) / kRows2Warps, kRows2Warps * 32, 0, st>>>(rp);
    c->launches++;
    OCT_CUDA(c, cudaGetLastError());
    return OCT_OK;
}

int oct_width2(oct_ctx* c, int64_t* out_dev, void* stream)
{
    if (!c || !out_dev) return OCT_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int rc = launch_anchors(c, nullptr, st, out_dev, 4);
    if (rc) return rc;
    RowsParams rp{};
    rp.latA = c->lat; rp.anchorA = c->anchorA(); rp.countersA = c->counters();
    rp.out = reinterpret_cast<unsigned long long*>(out_dev); rp.L = c->L;
    const uint32_t LW = c->L >> 2;
    launch_rows(kObsW2, rp, LW, st);
    c->launches++;
    OCT_CUDA(c, cudaGetLastError());
    return OCT_OK;
}

int oct_snapshot(oct_ctx* c, void* lattice_copy_dev, int64_t* anchor_out_dev, void* stream)
{
    if (!c || !lattice_copy_dev || !anchor_out_dev || (reinterpret_cast<uintptr_t>(lattice_copy_dev) & 15u)) return OCT_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    OCT_CUDA(c, cudaMemcpyAsync(lattice_copy_dev, c->lat, oct_lattice_bytes(c->L), cudaMemcpyDeviceToDevice, st));
    snapshot_anchor_kernel<<<1, 1, 0, st>>>(c->counters(), reinterpret_cast<long long*>(anchor_out_dev));
    c->launches++;
    OCT_CUDA(c, cudaGetLastError());
    return OCT_OK;
}

int oct_autocorr(oct_ctx* c, const void* snapshot_dev, const int64_t* snapshot_anchor_dev, int64_t* out_dev, void* stream)
{
    if (!c || !snapshot_dev || !snapshot_anchor_dev || !out_dev || (reinterpret_cast<uintptr_t>(snapshot_dev) & 15u)) return OCT_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int rc = launch_anchors(c, static_cast<const uint32_t*>(snapshot_dev), st, out_dev, 5);
    if (rc) return rc;
    RowsParams rp{};
    rp.latA = c->lat; rp.latB = static_cast<const uint32_t*>(snapshot_dev);
    rp.anchorA = c->anchorA(); rp.anchorB = c->anchorB(); rp.countersA = c->counters();
    rp.snapB = reinterpret_cast<const long long*>(snapshot_anchor_dev);
    rp.out = nullptr; rp.out_ch = reinterpret_cast<unsigned long long*>(out_dev); rp.L = c->L;   // C_h sums only: the kernel touches out_ch[0..4]
    const uint32_t LW = c->L >> 2;
    launch_rows(kObsCh, rp, LW, st);
    c->launches++;
    OCT_CUDA(c, cudaGetLastError());
    return OCT_OK;
}

int oct_slope_autocorr(oct_ctx* c, const void* snapshot_dev, int64_t* out_dev, void* stream)
{
    if (!c || !snapshot_dev || !out_dev || (reinterpret_cast<uintptr_t>(snapshot_dev) & 15u)) return OCT_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    OCT_CUDA(c, cudaMemsetAsync(out_dev, 0, 6 * sizeof(int64_t), st));
    const size_t n_vec = (size_t)c->L * c->L / 4 / 16;
    const size_t want = (n_vec + kSlopeThreads - 1) / kSlopeThreads;
    const unsigned blocks = (unsigned)(want < 148 * 16 ? want : 148 * 16);
    slope_autocorr_kernel<<<blocks, kSlopeThreads, 0, st>>>(reinterpret_cast<const uint4*>(c->lat), static_cast<const uint4*>(snapshot_dev),
                                                           n_vec, reinterpret_cast<unsigned long long*>(out_dev));
    c->launches++;
    OCT_CUDA(c, cudaGetLastError());
    return OCT_OK;
}

int oct_observe(oct_ctx* c, int what, const void* snapshot_dev, const int64_t* snapshot_anchor_dev, int64_t* out_dev, void* stream)
{
    if (!c || !out_dev || what <= 0 || what > (OCT_OBS_W2 | OCT_OBS_CH | OCT_OBS_CS)) return OCT_EINVAL;
    const bool need_snap = (what & (OCT_OBS_CH | OCT_OBS_CS)) != 0;
    if (need_snap && (!snapshot_dev || (reinterpret_cast<uintptr_t>(snapshot_dev) & 15u))) return OCT_EINVAL;
    if ((what & OCT_OBS_CH) && !snapshot_anchor_dev) return OCT_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int rc = OCT_OK;
    if (what & (OCT_OBS_W2 | OCT_OBS_CH)) rc = launch_anchors(c, (what & OCT_OBS_CH) ? static_cast<const uint32_t*>(snapshot_dev) : nullptr, st, out_dev, 16);
    else OCT_CUDA(c, cudaMemsetAsync(out_dev, 0, 16 * sizeof(int64_t), st));
    if (rc) return rc;
    RowsParams rp{};
    rp.latA = c->lat; rp.latB = static_cast<const uint32_t*>(snapshot_dev);
    rp.anchorA = c->anchorA(); rp.anchorB = c->anchorB(); rp.countersA = c->counters();
    rp.snapB = reinterpret_cast<const long long*>(snapshot_anchor_dev);
    rp.out = reinterpret_cast<unsigned long long*>(out_dev); rp.out_ch = rp.out + 4; rp.L = c->L;
    launch_rows(what, rp, c->L >> 2, st);
    c->launches++;
    OCT_CUDA(c, cudaGetLastError());
    return OCT_OK;
}

int oct_observe_batch(oct_ctx* const* cs, uint32_t n, int what, const void* const* snapshots_dev,
                      const int64_t* const* snapshot_anchors_dev, int64_t* out_dev, void* stream)
{
    if (!cs || n == 0 || !out_dev || what <= 0 || what > (OCT_OBS_W2 | OCT_OBS_CH | OCT_OBS_CS)) return OCT_EINVAL;
    const bool need_snap = (what & (OCT_OBS_CH | OCT_OBS_CS)) != 0, need_anchor = (what & (OCT_OBS_W2 | OCT_OBS_CH)) != 0;
    if (need_snap && !snapshots_dev) return OCT_EINVAL;
    if ((what & OCT_OBS_CH) && !snapshot_anchors_dev) return OCT_EINVAL;
    for (uint32_t i = 0; i < n; ++i) {
        if (!cs[i] || cs[i]->L != cs[0]->L) return OCT_EINVAL;
        if (need_snap && (!snapshots_dev[i] || (reinterpret_cast<uintptr_t>(snapshots_dev[i]) & 15u))) return OCT_EINVAL;
        if ((what & OCT_OBS_CH) && !snapshot_anchors_dev[i]) return OCT_EINVAL;
    }
    oct_ctx* c0 = cs[0];
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const uint32_t LW = c0->L >> 2;
    if (!need_anchor) OCT_CUDA(c0, cudaMemsetAsync(out_dev, 0, (size_t)n * 16 * sizeof(int64_t), st));
    ObsBatchParams bp{};
    bp.L = c0->L; bp.n_zero = 16;
    for (uint32_t m0 = 0; m0 < n; m0 += kMaxObsBatch) {
        const uint32_t nb = n - m0 < (uint32_t)kMaxObsBatch ? n - m0 : (uint32_t)kMaxObsBatch;
        for (uint32_t m = 0; m < nb; ++m) {
            const oct_ctx* c = cs[m0 + m];
            ObsMember& mb = bp.m[m];
            mb.latA = c->lat; mb.latB = need_snap ? static_cast<const uint32_t*>(snapshots_dev[m0 + m]) : nullptr;
            mb.anchorA = c->anchorA(); mb.anchorB = c->anchorB(); mb.colA = c->colA(); mb.colB = c->colB(); mb.blocksum = c->blocksum();
            mb.countersA = c->counters();
            mb.snapB = (what & OCT_OBS_CH) ? reinterpret_cast<const long long*>(snapshot_anchors_dev[m0 + m]) : nullptr;
            mb.out = reinterpret_cast<unsigned long long*>(out_dev) + (size_t)(m0 + m) * 16;
        }
        if (need_anchor) {
            const uint32_t nlat = (what & OCT_OBS_CH) ? 2u : 1u;
            const dim3 grid((LW + kColThreads - 1) / kColThreads, nlat, nb);
            column_gather_batch_kernel<<<grid, kColThreads, 0, st>>>(bp);
            column_anchor_batch_kernel<<<grid, kColThreads, 0, st>>>(bp);
            c0->launches += 2;
        }
        launch_rows_batch(what, bp, nb, LW, st);
        c0->launches++;
        OCT_CUDA(c0, cudaGetLastError());
    }
    return OCT_OK;
}

int oct_fetch(oct_ctx* c, const void* src_dev, void* dst_host, size_t bytes, void* stream)
{
    if (!c || !src_dev || !dst_host) return OCT_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    OCT_CUDA(c, cudaMemcpyAsync(dst_host, src_dev, bytes, cudaMemcpyDeviceToHost, st));
    OCT_CUDA(c, cudaStreamSynchronize(st));
    return OCT_OK;
}

int oct_export(oct_ctx* c, void* lattice_host, void* stream)
{
    if (!c || !lattice_host) return OCT_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    OCT_CUDA(c, cudaMemcpyAsync(lattice_host, c->lat, oct_lattice_bytes(c->L), cudaMemcpyDeviceToHost, st));
    OCT_CUDA(c, cudaStreamSynchronize(st));
    return OCT_OK;
}

int oct_upload(oct_ctx* c, const void* lattice_host, void* stream)
{
    if (!c || !lattice_host) return OCT_EINVAL;
    OCT_CUDA(c, cudaMemcpyAsync(c->lat, lattice_host, oct_lattice_bytes(c->L), cudaMemcpyHostToDevice,
                                static_cast<cudaStream_t>(stream)));
    return OCT_OK;
}

int oct_counters(oct_ctx* c, int64_t* out_host, void* stream)
{
    if (!c || !out_host) return OCT_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    unsigned long long tmp[2];
    OCT_CUDA(c, cudaMemcpyAsync(tmp, c->counters(), sizeof(tmp), cudaMemcpyDeviceToHost, st));
    OCT_CUDA(c, cudaStreamSynchronize(st));
    out_host[0] = (int64_t)tmp[1];   // h(0,0)
    out_host[1] = (int64_t)tmp[0];   // net
    return OCT_OK;
}

int oct_mcs(const oct_ctx* c, uint64_t* t_out)
{
    if (!c || !t_out) return OCT_EINVAL;
    *t_out = c->t;
    return OCT_OK;
}

int oct_launch_count(const oct_ctx* c, uint64_t* n_out)
{
    if (!c || !n_out) return OCT_EINVAL;
    *n_out = c->launches;
    return OCT_OK;
}

int oct_destroy(oct_ctx* c)
{
    if (!c) return OCT_EINVAL;
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->aux) cudaStreamDestroy(c->aux);
    delete c;
    return OCT_OK;
}

const char* oct_strerror(int code)
{
    switch (code) {
        case OCT_OK: return "ok";
        case OCT_EINVAL: return "invalid argument";
        case OCT_ECUDA: return "CUDA error (see oct_last_error)";
        case OCT_ENOMEM: return "out of host memory";
        case OCT_ESTATE: return "invalid state";
        case OCT_ETOOBIG: return "lattice larger than the fixed scratch of oct_width2_static (L <= 65536)";
        default: return "unknown error code";
    }
}

const char* oct_last_error(const oct_ctx* c) { return c ? c->last_error.c_str() : ""; }

double oct_w2_from_sums(uint32_t L, int64_t S1, int64_t S2)
{
    const __int128 N = (__int128)L * L;
    const __int128 num = N * (__int128)S2 - (__int128)S1 * (__int128)S1;
    return (double)((long double)num / ((long double)N * (long double)N));
}

double oct_c_from_sums(uint32_t L, int64_t St, int64_t Ss, int64_t Sts)
{
    const __int128 N = (__int128)L * L;
    const __int128 num = N * (__int128)Sts - (__int128)St * (__int128)Ss;
    return (double)((long double)num / ((long double)N * (long double)N));
}

double oct_cs_from_sums(uint64_t M, int64_t n11, int64_t n1t, int64_t n1s)
{
    if (M == 0) return 0.0;
    const __int128 m = (__int128)M;
    const __int128 num = m * (__int128)n11 - (__int128)n1t * (__int128)n1s;
    return (double)((long double)num / ((long double)m * (long double)m));
}

double oct_time_per_sweep(uint32_t L, int scheme)
{
    if (check_scheme(L, scheme) != OCT_OK) return 0.0;
    const SchemeFields f = split_scheme(scheme);
    if (f.dev <= OCT_DEV_DT) return 1.0;
    const double D = (double)(1u << f.log2D), w = (double)f.width();
    return ((D - w) / D) * ((D - w) / D);   // Eq. (9) :137 with reading R9
}

}  // extern "C"

// oct_width2_static: the W^2 sums of oct_width2 (Eq. (3)) for a caller that has a packed lattice and an
// output buffer on the device and NOTHING ELSE -- no handle, no workspace, and no way to get either.
//
// Who that is.  Every other entry point of this library works on a handle whose workspace the caller allocated
// (oct_workspace_bytes).  Some users of the lattice cannot do that:
//   * a measurement hook inside somebody else's simulation loop, which is handed the lattice pointer and a slot for the
//     result and does not own a device allocator (the host program has given all of HBM to its lattices: one L = 2^17
//     lattice is 4 GiB, an ensemble fills the card);
//   * code that runs while other streams of the process are busy sweeping: cudaMalloc / cudaFree synchronise the whole
//     device, so an allocation made for one measurement would stall every concurrent replica;
//   * code in a section of the host program where allocating is forbidden outright (a real-time loop, a callback that
//     may not call the allocator, a process running under a fixed memory budget that is already spent).
// For them the scratch of the reduction -- column 0 gathered into a compact array, the net slope of every CTA's part of
// it, the row anchors h(0,y) - h(0,0), and the two counters the reduction copies into its output -- lives in ONE
// file-scope __device__ array of this translation unit, sized for L <= OCT_WIDTH2_STATIC_MAX_L.  The array is part of
// the library image: every GPU on which the library is loaded holds its ~321 KiB from module load until the process
// exits, whether or not this entry point is ever called.  This file calls no cudaMalloc, cudaFree, cudaMemset or any
// library routine that allocates; the three launches below are all the device work there is.
//
// The kernels are the ones oct_width2 runs (the same device bodies from observe.cuh / observe_rows.cuh, so the sums are
// the same integers), wrapped so that their scratch pointers come from the static array.
//
// What a host-side name of a __device__ array is.  In host code `g_width2_scratch` is a stand-in object of the host
// linker, not a device address: handing it (or &g_width2_scratch[0]) to a kernel gives the kernel a HOST address, which
// faults -- or, on a system where the GPU can reach host memory, silently reads and writes the wrong memory.  The
// device address is what cudaGetSymbolAddress returns, per device, with that device current.  scratch_on_current_device()
// below asks for it once per device and keeps it.
#include <cstdint>
#include <mutex>

#include <cuda_runtime.h>

#include "../../include/oct.h"
#define OCT_OBSERVE_BODIES_ONLY   // device bodies and parameter blocks only: the kernels of observe.cuh live in oct_api.cu
#include "observe.cuh"
#include "observe_rows.cuh"

using namespace octb;

namespace {

constexpr uint32_t kStaticMaxL = OCT_WIDTH2_STATIC_MAX_L;
static_assert((kStaticMaxL & (kStaticMaxL - 1)) == 0 && kStaticMaxL / 4 <= (uint32_t)kColThreads * kColMaxBlocks, "static maximum");

// Layout of the scratch, in bytes.  The offsets do not depend on the L of a call.
constexpr size_t kOffCounters = 0;                                   // 2 x uint64 {net, h(0,0)}: what rows3_body copies to out[3], out[2]
constexpr size_t kOffBlocksum = 256;                                 // kColMaxBlocks x int32: net sigma_y of each CTA's part of column 0
constexpr size_t kOffAnchor   = 1024;                                // L x int32: h(0,y) - h(0,0)
constexpr size_t kOffColumn   = kOffAnchor + 4 * (size_t)kStaticMaxL; // L/4 words: column 0 of the packed lattice, compact
constexpr size_t kScratchBytes = kOffColumn + kStaticMaxL;            // 1024 + 5 L_max = 328 704 bytes
static_assert(kOffBlocksum + sizeof(int32_t) * kColMaxBlocks <= kOffAnchor, "blocksum overlaps anchors");

static __device__ __align__(256) unsigned char g_width2_scratch[kScratchBytes];

// ---- the kernels: oct_width2's three launches, with their scratch at fixed offsets of `scratch` ---------------------------
// `scratch` is the DEVICE address of g_width2_scratch (device code could also name the array directly; it is passed so
// that the kernels say which memory they use).

// gathers column 0 and every CTA's net slope; CTA 0 also deposits the caller's (net, h00) where the reduction reads them
__global__ void __launch_bounds__(kColThreads)
width2_static_gather_kernel(const uint32_t* __restrict__ lat, uint32_t L, unsigned char* __restrict__ scratch, long long h00, long long net)
{
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        unsigned long long* counters = reinterpret_cast<unsigned long long*>(scratch + kOffCounters);
        counters[0] = (unsigned long long)net;
        counters[1] = (unsigned long long)h00;
    }
    column_gather_body(lat, L, reinterpret_cast<uint32_t*>(scratch + kOffColumn), reinterpret_cast<int32_t*>(scratch + kOffBlocksum));
}

// row anchors from the gathered column; also clears out[0..3], the accumulators of the reduction that follows
__global__ void __launch_bounds__(kColThreads)
width2_static_anchor_kernel(unsigned char* __restrict__ scratch, uint32_t L, unsigned long long* __restrict__ out)
{
    column_anchor_body(reinterpret_cast<const uint32_t*>(scratch + kOffColumn), reinterpret_cast<const int32_t*>(scratch + kOffBlocksum), L,
                       reinterpret_cast<int32_t*>(scratch + kOffAnchor), out, 4);
}

// the reduction itself: rows3_body<kObsW2> (one warp per word-row), anchors and counters read from the scratch
template <int RUN>
__global__ void __launch_bounds__(kRows2Warps * 32)
width2_static_rows_kernel(const uint32_t* __restrict__ lat, uint32_t L, const unsigned char* __restrict__ scratch, unsigned long long* __restrict__ out)
{
    RowsParams P;
    P.latA = lat; P.latB = nullptr;
    P.anchorA = reinterpret_cast<const int32_t*>(scratch + kOffAnchor); P.anchorB = nullptr;
    P.countersA = reinterpret_cast<const unsigned long long*>(scratch + kOffCounters);
    P.snapB = nullptr; P.heights = nullptr; P.out = out; P.out_ch = nullptr; P.L = L;
    rows3_body<kObsW2, RUN>(P);
}

// ---- set-up: the device address of the scratch, once per device ---------------------------------------------------------
constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
unsigned char* g_scratch_dev[kMaxDevices];   // [d] = device address of g_width2_scratch on device d, nullptr until first use there

// The first call on a device asks the runtime for the array's address on THAT device (it must be the current one: the
// symbol is looked up in the current device's copy of the module) and checks the answer; later calls reuse it.
int scratch_on_current_device(unsigned char** out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return OCT_ECUDA;
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_dev[dev]) {
        int major = 0;
        if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess || major != 10) return OCT_ECUDA;
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_width2_scratch);
        if (e != cudaSuccess || !p) return OCT_ECUDA;
        g_scratch_dev[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_scratch_dev[dev];
    return OCT_OK;
}

}  // namespace

extern "C" int oct_width2_static(const void* lattice_dev, uint32_t L, int64_t h00, int64_t net, int64_t* out_dev, void* stream)
{
    if (!lattice_dev || !out_dev) return OCT_EINVAL;
    if ((reinterpret_cast<uintptr_t>(lattice_dev) & 15u) || (reinterpret_cast<uintptr_t>(out_dev) & 7u)) return OCT_EINVAL;
    if (L < 16u || L > (1u << 17) || (L & (L - 1u)) != 0u) return OCT_EINVAL;   // not a lattice size of this library at all
    if (L > kStaticMaxL) return OCT_ETOOBIG;                 // before any CUDA call: nothing is enqueued, nothing is touched
    unsigned char* scratch = nullptr;
    const int rc = scratch_on_current_device(&scratch);
    if (rc != OCT_OK) return rc;

    // Nothing in the scratch has to start at zero: every byte a call reads (counters, blocksum[0 .. CTAs), column[0 .. L/4),
    // anchor[0 .. L)) is written earlier in the same call, and what a previous, larger call left beyond those ranges is
    // never read.  The only accumulators are out[0] and out[1]; the anchor kernel clears out[0..3] before the reduction adds.
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const uint32_t LW = L >> 2;
    const unsigned col_blocks = (LW + kColThreads - 1) / kColThreads;
    const uint32_t* lat = static_cast<const uint32_t*>(lattice_dev);
    unsigned long long* out = reinterpret_cast<unsigned long long*>(out_dev);
    width2_static_gather_kernel<<<col_blocks, kColThreads, 0, st>>>(lat, L, scratch, (long long)h00, (long long)net);
    width2_static_anchor_kernel<<<col_blocks, kColThreads, 0, st>>>(scratch, L, out);
    const unsigned row_blocks = (LW + kRows2Warps - 1) / kRows2Warps;
    if (LW >= 512u) width2_static_rows_kernel<16><<<row_blocks, kRows2Warps * 32, 0, st>>>(lat, L, scratch, out);
    else            width2_static_rows_kernel<4><<<row_blocks, kRows2Warps * 32, 0, st>>>(lat, L, scratch, out);
    return cudaGetLastError() == cudaSuccess ? OCT_OK : OCT_ECUDA;
}

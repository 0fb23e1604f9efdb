/*
 * oct.h -- C ABI of liboct_b200: the domain-decomposed (DD) random-sequential sweep of the 2+1-d
 * octahedron model of arXiv 1705.01022 (Kelling, Odor, Gemming) on one NVIDIA B200 (sm_100a), with
 * height reconstruction and the exact integer sums for W^2(t) and C_h(t,s).
 *
 * Citations are PAPER.md line numbers plus the section / equation they fall in; "R<n>" are the
 * readings of silent or garbled passages listed in DESIGN.md.
 *
 * GENERAL RULES
 *  - Every function returns OCT_OK (0) or a negative error code; nothing throws, aborts or prints.
 *  - Pointers named *_dev are DEVICE pointers, *_host are HOST pointers.  The caller owns every device
 *    buffer and the stream; the library never allocates device memory.  `stream` is a cudaStream_t
 *    passed as void* (NULL = the legacy default stream).
 *  - Unless stated otherwise a call only ENQUEUES work on `stream` and returns; results land in
 *    device buffers in stream order.  Calls that touch host buffers say whether they synchronise.
 *  - ONE STREAM PER HANDLE at a time: the observables share scratch in the handle's workspace (the column
 *    anchors), so calls on one handle must be ordered (same stream, or the caller's events).  Different
 *    handles are independent and may run on different streams concurrently.
 *  - One process may drive several GPUs: a handle belongs to the device that was current at oct_create (its buffers
 *    live there); make that device current again for every call on the handle.  Nothing is cached across devices.
 *  - The library runs on the current CUDA device and requires compute capability 10.x; there is no
 *    CPU fallback: without a usable device every compute call returns OCT_ECUDA.
 *  - Determinism: the lattice after oct_sweep depends only on (L, seed, init, the sequence of
 *    (n_mcs, p, q, scheme)); never on grid size, timing or GPU model.  All randomness is counter-based
 *    Philox4x32-10 keyed by (seed, mcs, set, domain, cell, step) (R19).
 *
 * DATA FORMATS
 *  - Site (x,y), 0 <= x,y < L, periodic (:127).  sigma_x(x,y) = h(x,y)-h(x-1,y) and
 *    sigma_y(x,y) = h(x,y)-h(x,y-1), each +-1, stored AT site (x,y) as one bit (1 <=> +1)  (:140, R2/R3).
 *  - Packed lattice (:166, R4): L*L/4 bytes, little-endian uint32 words, word index wy*(L/4)+wx holds
 *    the 4x4 sites (4wx+i, 4wy+j); sigma_x at bit 2(4j+i), sigma_y at bit 2(4j+i)+1.  This is both the
 *    device layout and the exchange ("canonical") layout.
 *  - Heights: int32, row-major [y*L + x].
 */
#ifndef OCT_B200_H
#define OCT_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct oct_ctx oct_ctx;   /* opaque host-side handle, owned by the library until oct_destroy */

enum { OCT_OK = 0, OCT_EINVAL = -1, OCT_ECUDA = -2, OCT_ENOMEM = -3, OCT_ESTATE = -4,
       OCT_ETOOBIG = -5   /* oct_width2_static only: L is valid but beyond that call's fixed scratch */ };

enum {
    OCT_INIT_FLAT = 0,          /* h = (x+y)&1: every word 0x33CC33CC, W^2 = 1/4 (R5)               */
    OCT_INIT_FLAT_SHIFTED = 1,  /* h = -((x+y)&1): the bitwise complement, every word 0xCC33CC33     */
    OCT_INIT_FROM_DEVICE = 2    /* the caller already filled lattice_dev (canonical words)          */
};

/* scheme = dev | blk<<4 | tcx<<8 | tcy<<12 | log2D<<16 | ka<<21 | w<<23      (notation of Sec. 3.1.1 :176-182)
 *   dev  (device layer, Sec. 3 :129-150):  0 DTr  double tiling with random origin   (:148-150)
 *                                          1 DT   double tiling, fixed origin         (:142-146)
 *                                          2 DB   dead border, free origin, width 5   (:133-140, :166)
 *                                          3 cDB  dead border, origin on the 4-site grid, width 1 (:166)
 *                                          4 DBh  DB with t_async = 1/2 MCS: two intervals per sweep, each with
 *                                                 its own origin and half of the collective steps (:204-206, R27)
 *   blk  (block layer, single-hit, Sec. 3.1 :168-174):
 *                                          0 DB   random cell origin per collective step; "ignoring
 *                                                 borders" when only one of p,q is non-zero, delayed
 *                                                 borders otherwise (:174, R16)
 *                                          1 DB   delayed borders forced
 *                                          2 DT   one random quadrant of every cell per step (:170)
 *                                          3 DTr  DT whose cell origin also moves every step ("DTrDTr", :234, R26)
 *   tcx,tcy: log2 of the thread-cell edge in words of 4 sites, "TC=tcx,tcy" (:180); cell = 4<<tc sites
 *   log2D  : log2 of the device-layer domain edge D in sites (the sub-tile one worker sweeps)
 *   ka     : dead-border layers DB / cDB only: t_async = 2^-ka MCS, ka = 0, 1, 2 -- one sweep is 2^ka asynchronous
 *            intervals, each with its own origin and 1/2^ka of the collective steps (:204-206, R27; DBh == DB with ka = 1)
 *   w      : DB / cDB only: dead-border width in sites, 1..7; 0 = the scheme's own (DB 5, cDB 1).  DB with w = 1 is the
 *            "DB with a border-width of one lattice site" and a free origin of :208; the paper's bit-coded kernel needs 5
 *            there because tiles share 4x4-site words (:166) -- here words shared by two tiles are written back bit-wise  */
#define OCT_SCHEME(dev, blk, tcx, tcy, log2D) \
    ((dev) | ((blk) << 4) | ((tcx) << 8) | ((tcy) << 12) | ((log2D) << 16))
#define OCT_SCHEME_DB(dev, blk, tcx, tcy, log2D, ka, w) (OCT_SCHEME(dev, blk, tcx, tcy, log2D) | ((ka) << 21) | ((w) << 23))
enum { OCT_DEV_DTR = 0, OCT_DEV_DT = 1, OCT_DEV_DB = 2, OCT_DEV_CDB = 3, OCT_DEV_DBH = 4 };
enum { OCT_BLK_DB = 0, OCT_BLK_DB_DELAYED = 1, OCT_BLK_DT = 2, OCT_BLK_DTR = 3 };

/* Sizes of the caller-allocated device buffers for an L x L lattice (0 if L is invalid). */
size_t oct_lattice_bytes(uint32_t L);      /* L*L/4                                                  */
size_t oct_workspace_bytes(uint32_t L);    /* 1280 + 10 L: counters, two arrays of row anchors, column scratch */

/* Create a simulation on caller-owned device buffers (both 16-byte aligned).  Problem statement:
 * Sec. 2.1 :25-34 (model), :127 (periodic, L x L).  L must be a power of two, 16 <= L <= 2^17.
 * init = FLAT / FLAT_SHIFTED enqueue a fill of lattice_dev; FROM_DEVICE leaves it untouched.  The
 * device counters (net deposits, tracked h(0,0)) are zeroed; the MCS clock starts at 0.
 * Errors: EINVAL (bad L / init / null pointer), ECUDA (no sm_100 device, launch failure), ENOMEM. */
int oct_create(oct_ctx** out, uint32_t L, uint64_t seed, int init,
               void* lattice_dev, void* workspace_dev, void* stream);

/* Overwrite the clock and the tracked anchors (used with INIT_FROM_DEVICE / oct_upload when the
 * lattice is a continuation of an earlier run).  t < 2^32. */
int oct_set_state(oct_ctx*, uint64_t t_mcs, int64_t h00, int64_t net, void* stream);

/* n_mcs sweeps of the whole lattice (1 MCS = L^2 update attempts, :106) under DD scheme `scheme`,
 * deposition probability p at local minima and removal probability q at local maxima (Eq. (1)
 * :27-34; p,q in [0,1], quantised to 1/65536, R18).  DTr/DT: 4 kernel launches per MCS, one per domain
 * set, in the permutation drawn for that MCS (:144); DB/cDB: 2^ka launches per sweep (DBh: 2), and one such sweep
 * lasts (1 - N_border/N) MCS of physical time (Eq. (9) :137, R9; see oct_time_per_sweep).
 * oct_sweep(a) followed by oct_sweep(b) equals oct_sweep(a+b).
 * Errors (nothing is enqueued): EINVAL for p,q outside [0,1], unknown dev/blk, cell larger than the
 * domain, blk=DT/DTr with tc<1 (:182), L < 2D for DT/DTr (2D x 2D tiles) or L < D for the dead-border layers,
 * D outside {32,64,128,256} or a (D,TC) pair the library was not built for, t+n_mcs > 2^32-1.
 * ECUDA: a launch failed (text via oct_last_error); the sweeps enqueued before the failing one stay enqueued and
 * oct_mcs() reports how many were. */
int oct_sweep(oct_ctx*, uint64_t n_mcs, double p, double q, int scheme, void* stream);

/* The same n_mcs sweeps on n independent simulations of ONE lattice size at once (ensembles: the paper's curves are
 * means over n = 20 ... 4367 runs, many at L <= 2^13): every kernel launch covers the
 * domains of all members (grid = domains x members, at most 256 members per launch), so small lattices fill the
 * GPU.  Each member keeps its own lattice, counters, seed and clock; its result is bit-identical to what
 * oct_sweep on that handle alone would give.  The two halves of the ensemble run side by side -- one on `stream`, one on
 * a helper stream of handle 0 that forks from `stream` and joins it again before the call returns -- so that the last
 * domains of one half's launch overlap the other half's next launch; for the caller everything is ordered on `stream`.
 * Shapes without a many-lattices kernel (D = 128 other than TC=1,1, every D = 256 shape, the bit-packed kernel) run the
 * members one after the other.  The kernel option of handle 0 applies.
 * Errors: as oct_sweep, plus EINVAL for n = 0, a null or repeated handle, or members of different L.  A CUDA failure
 * between two MCS returns ECUDA with every member's clock at the sweeps completed (as oct_sweep).  A failure INSIDE an
 * MCS -- some launches of its domain sets enqueued, others not -- returns ESTATE: the members' lattices then hold a partly
 * swept MCS that no clock value describes; re-create or re-upload them (oct_last_error(handles[0]) has the CUDA text). */
int oct_sweep_batch(oct_ctx* const* handles, uint32_t n, uint64_t n_mcs, double p, double q, int scheme, void* stream);

/* Integrate the slopes into int32 heights h[y*L+x] (:52 "peaks of the octahedra define the height
 * profile"; anchor h(0,0) tracked exactly, R20).  heights_dev holds L*L int32. */
int oct_heights(oct_ctx*, int32_t* heights_dev, void* stream);

/* Integer sums for the roughness W^2(L,t) of Eq. (3) :61 (R6): out_dev[4] = {S1, S2, c, net} with
 * c = h(0,0), S1 = sum (h-c), S2 = sum (h-c)^2 over all sites, net = deposits - removals so far.
 * Exact as long as L^2 * max (h-c)^2 < 2^63. */
int oct_width2(oct_ctx*, int64_t* out_dev, void* stream);

/* oct_width2 WITHOUT a handle and without a workspace: the same sums, out_dev[4] = {S1, S2, c, net} (Eq. (3) :61, R6),
 * of the packed lattice at lattice_dev (canonical words, 16-byte aligned, L x L sites), with c = h00 and net passed
 * in by value and copied through to out_dev[2], out_dev[3] (W^2 does not depend on c; pass 0, 0 if you do not track them).
 *
 * For callers that cannot allocate device memory at all, not even the workspace every other call needs: a measurement
 * hook that is handed a lattice and a result slot by a program that owns all of HBM; code that must not call cudaMalloc /
 * cudaFree because those synchronise the whole device and would stall the replicas sweeping on other streams; code in a
 * part of the host program where allocation is forbidden or the memory budget is spent.  This call allocates nothing,
 * on the device or through any library: its scratch (column 0 gathered, per-CTA net slopes, the L row anchors, two
 * counters) is a fixed array inside the library image, 1024 + 5 * OCT_WIDTH2_STATIC_MAX_L = 328 704 bytes, which every
 * GPU that loads the library holds until the process exits.
 *
 * LIMIT: 16 <= L <= OCT_WIDTH2_STATIC_MAX_L (2^16), a power of two.  A valid but larger L (2^17) returns OCT_ETOOBIG
 * ("lattice larger than the fixed scratch of oct_width2_static"); nothing is enqueued and no memory is touched.
 * FIRST CALL ON A DEVICE: looks up the device address of the array on the current device (cudaGetSymbolAddress, result
 * checked, kept per device); make that first call with the right device current and before any stream capture begins.
 * SHARED SCRATCH: all calls on one device use the same array, which keeps whatever the last call left.  That is
 * harmless for calls that follow each other (each call writes every byte it later reads, and clears out_dev[0..3]
 * itself), but two calls that can overlap on the GPU -- different streams, or different host threads without a common
 * stream -- race on it and give garbage: put them on one stream or order them with events.
 * Only ENQUEUES three launches on `stream`.  Results are the integers oct_width2 gives for the same lattice.
 * Errors: EINVAL (null / misaligned pointer, L not a power of two or < 16), ETOOBIG, ECUDA (no sm_100 device, the symbol
 * look-up or a launch failed). */
#define OCT_WIDTH2_STATIC_MAX_L 65536u
int oct_width2_static(const void* lattice_dev, uint32_t L, int64_t h00, int64_t net, int64_t* out_dev, void* stream);

/* Waiting-time snapshot for aging (:75-80): copies the packed lattice to lattice_copy_dev
 * (oct_lattice_bytes, 16-byte aligned) and writes anchor_out_dev[2] = {h(0,0), net} at this moment. */
int oct_snapshot(oct_ctx*, void* lattice_copy_dev, int64_t* anchor_out_dev, void* stream);

/* Integer sums for the height autocorrelation C_h(t,s) of Eq. (6) :92-98 (R7) between the current
 * lattice and a snapshot: out_dev[5] = {S_t, S_s, S_ts, c_t, c_s}, S_t = sum (h_t-c_t),
 * S_s = sum (h_s-c_s), S_ts = sum (h_t-c_t)(h_s-c_s).  With snapshot == current state the sums
 * reproduce oct_width2's (C_h(s,s) = W^2(s), :97).  snapshot_dev must be 16-byte aligned (EINVAL otherwise). */
int oct_autocorr(oct_ctx*, const void* snapshot_dev, const int64_t* snapshot_anchor_dev,
                 int64_t* out_dev, void* stream);

/* Integer sums for the slope (lattice-gas) autocorrelation C_s(t,s) of PAPER.md:85-88 between the current
 * lattice and a snapshot (oct_snapshot's lattice copy, 16-byte aligned), n = slope bit:
 * out_dev[6] = {sum nx_t nx_s, sum ny_t ny_s, sum nx_t, sum ny_t, sum nx_s, sum ny_s} (x and y slopes apart;
 * the four single sums are L*L/2 for any valid surface).  C_s = oct_cs_from_sums over M = 2 L^2 variables
 * (or M = L^2 for one direction); C_s(s,s) = 1/4. */
int oct_slope_autocorr(oct_ctx*, const void* snapshot_dev, int64_t* out_dev, void* stream);

/* ONE pass over the current lattice (and the snapshot) for any combination `what` of the observables above:
 * OCT_OBS_W2 (oct_width2's sums), OCT_OBS_CH (oct_autocorr's), OCT_OBS_CS (oct_slope_autocorr's).  A measurement point
 * of an aging run wants all three: together they read the lattice and the snapshot once (2 x L^2/4
 * bytes) instead of five times.  out_dev[16] (int64; all of it is overwritten):
 *   [0..3] = {S1, S2, c, net}   [4..8] = {S_t, S_s, S_ts, c_t, c_s}   [9..14] = {xx, yy, x_t, y_t, x_s, y_s}   [15] = 0
 * with the meanings given at oct_width2 / oct_autocorr / oct_slope_autocorr; groups not asked for stay zero.
 * snapshot_dev (16-byte aligned) is needed for CH and CS, snapshot_anchor_dev for CH; EINVAL otherwise. */
enum { OCT_OBS_W2 = 1, OCT_OBS_CH = 2, OCT_OBS_CS = 4 };
int oct_observe(oct_ctx*, int what, const void* snapshot_dev, const int64_t* snapshot_anchor_dev,
                int64_t* out_dev, void* stream);

/* oct_observe for n simulations of ONE lattice size in as many launches as for one (three per 64 members): a measurement
 * point of an ensemble run.  snapshots_dev / snapshot_anchors_dev are HOST arrays of n device
 * pointers (member i's oct_snapshot buffers; may be NULL when `what` needs none); out_dev holds n x 16 int64, member i's
 * sums at out_dev + 16 i with the layout of oct_observe.  Results are identical to n oct_observe calls.
 * Errors: as oct_observe, plus EINVAL for n = 0, a null handle or members of different L. */
int oct_observe_batch(oct_ctx* const* handles, uint32_t n, int what, const void* const* snapshots_dev,
                      const int64_t* const* snapshot_anchors_dev, int64_t* out_dev, void* stream);

/* Copy `bytes` bytes of a device buffer (e.g. the sums above) to host memory.  SYNCHRONISES `stream`. */
int oct_fetch(oct_ctx*, const void* src_dev, void* dst_host, size_t bytes, void* stream);

/* Copy the packed lattice device -> host (canonical words).  SYNCHRONISES `stream`. */
int oct_export(oct_ctx*, void* lattice_host, void* stream);
/* Copy a packed lattice host -> device (enqueued; the host buffer must stay valid until the stream
 * reaches the copy; pinned memory makes it asynchronous).  Anchors/clock are NOT changed. */
int oct_upload(oct_ctx*, const void* lattice_host, void* stream);
/* Read the device counters: out_host[2] = {h(0,0), net}.  SYNCHRONISES `stream`. */
int oct_counters(oct_ctx*, int64_t* out_host, void* stream);

int oct_mcs(const oct_ctx*, uint64_t* t_out);           /* sweeps done so far                        */
int oct_destroy(oct_ctx*);                              /* frees the handle only (buffers are yours) */
const char* oct_strerror(int code);
const char* oct_last_error(const oct_ctx*);             /* text of the last CUDA failure, or ""     */

/* Implementation options.  They never change results (every kernel is bit-identical to the oracle), only
 * which kernel runs.  OCT_OPT_KERNEL: AUTO picks the link-entry kernel (one entry of four or two link bytes per site
 * in shared memory, no atomics) wherever one is built (every accepted (D, TC) except D = 32 with TC=2,2) and the bit-packed
 * kernel otherwise; BITPACKED forces the latter; LINKS_B selects the alternative work split (another number of
 * warps per domain) or entry size (four link bytes per site instead of two, for TC=2,2) where one is built.
 * EINVAL for unknown options / values. */
enum { OCT_OPT_KERNEL = 1 };
enum { OCT_KERNEL_AUTO = 0, OCT_KERNEL_BITPACKED = 1, OCT_KERNEL_LINKS_B = 2 };
int oct_set_option(oct_ctx*, int option, int value);

/* Number of kernel launches the library has enqueued through this handle (for bench accounting). */
int oct_launch_count(const oct_ctx*, uint64_t* n_out);

/* Pure host helpers (no device work). */
double oct_w2_from_sums(uint32_t L, int64_t S1, int64_t S2);                    /* (N*S2 - S1^2)/N^2  */
double oct_c_from_sums(uint32_t L, int64_t St, int64_t Ss, int64_t Sts);        /* (N*Sts - St*Ss)/N^2 */
double oct_cs_from_sums(uint64_t M, int64_t n11, int64_t n1t, int64_t n1s);     /* (M*n11 - n1t*n1s)/M^2 */
double oct_time_per_sweep(uint32_t L, int scheme);   /* 1 for DT/DTr; (1 - N_border/N) = ((D-w)/D)^2 for DB/cDB/DBh (R9) */
int    oct_scheme_supported(uint32_t L, int scheme); /* OCT_OK or OCT_EINVAL, same checks as oct_sweep */

#ifdef __cplusplus
}
#endif
#endif /* OCT_B200_H */

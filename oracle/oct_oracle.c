/*
 * oct_oracle.c -- CPU ORACLE for the octahedron-model sweep of arXiv 1705.01022.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Plain, slow, single-threaded C that follows the
 * paper and the readings listed in DESIGN.md step by step.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.  It shares
 * no code, header, table or constant generator with the CUDA path under paper_1705_01022_b200/.
 *
 * What each part follows (PAPER.md line : section):
 *   - update rule                      Eq. (1) :27-34, Fig. 1 caption :50, :52, :140   -> orc_attempt
 *   - true random-sequential dynamics  :15/:44, 1 MCS = L^2 attempts :106               -> orc_sweep_rs
 *   - device-layer DD: DB/cDB          Sec. 3.0.1 :133-140, :166; t_async = 1/2^k :204-206, border width :202 -> orc_sweep_dd
 *                      DT, DTr         Sec. 3.0.2 :142-146, Sec. 3.0.3 :148-150          -> orc_sweep_dd
 *   - block-layer single-hit DB / DT   Sec. 3.1 :168-174; DT with moving origin (DTr) :234 -> domain_sweep
 *   - roughness W^2, autocorr C_h      Eq. (3) :61, Eq. (6) :92-98                       -> orc_sums, orc_autocorr_sums
 *   - slope (lattice-gas) autocorr C_s :85-88 (unnumbered equation before Eq. (6))       -> orc_slope_autocorr_sums
 *   - RNG (paper silent)               Philox4x32-10, Salmon et al. SC'11; keying = DESIGN.md R19
 *
 * Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): Philox known-answer vectors and cuRAND's host
 * implementation; flat-state constants; brute-force of the height definition on the 4x4 lattice;
 * row/column conservation and curl-freeness; tracked vs recomputed heights (two paths); order
 * independence of every DD phase; complement symmetry; split invariance; attempt-trace properties
 * (coverage, uniformity, cell geometry); W^2(0)=1/4; C_h(s,s)=W^2(s); C_s(s,s)=1/4, C_s against the
 * complement = -1/4 and against slopes taken straight from a height array; KPZ growth exponent band.
 * Absolute W^2(t)/C(t,s) curves of the paper are figures only: "parity unpinned" against those.
 *
 * Conventions.  Site (x,y), 0 <= x,y < L, periodic.  sigma_x(x,y) = h(x,y)-h(x-1,y),
 * sigma_y(x,y) = h(x,y)-h(x,y-1), both +-1, stored AT site (x,y), bit 1 <=> +1 (:140 "one slope is
 * encoded on-site (to the left neighbor)").  Canonical packing (:166 "each 32-bit word encodes 4x4
 * lattice sites"): word wy*(L/4)+wx holds sites (4wx+i, 4wy+j); sigma_x at bit 2(4j+i), sigma_y at
 * bit 2(4j+i)+1.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------------------------------ RNG */

/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  round(c,k) = (hi(M1*c2)^c1^k0, lo(M1*c2),
 * hi(M0*c0)^c3^k1, lo(M0*c0)); key bumped by (W0,W1) between rounds; 10 rounds. */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)M0 * c0;
        uint64_t p1 = (uint64_t)M1 * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        if (r < 9) { k0 += W0; k1 += W1; }
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Stream tags (R19): counter = (c0, c1, tag<<30 | set<<28 | dom, t). */
enum { TAG_CELL = 0, TAG_BLOCK = 1, TAG_GLOBAL = 2, TAG_RS = 3 };

/* ---------------------------------------------------------------------------------------- state */

typedef struct orc_trace_rec {   /* one record per update attempt (test hook) */
    uint32_t x, y;               /* global site */
    uint32_t t, set, dom, k, cell;
    int32_t  cls;                /* block-layer DB class 0/1/2, -1 for DT / RS */
    int32_t  result;             /* +1 deposited, -1 removed, 0 nothing, 2 discarded by dead border */
} orc_trace_rec;

typedef struct orc_state {
    uint32_t L;
    uint64_t seed;
    uint64_t t;          /* sweeps done (absolute MCS index of the next sweep) */
    int64_t  net;        /* deposits minus removals */
    int64_t  h00;        /* tracked height of site (0,0) */
    uint32_t *lat;       /* (L/4)^2 canonical words */
    int32_t  *h;         /* incrementally tracked heights, or NULL */
    /* test hooks */
    uint64_t shuffle;    /* != 0: visit domains of a set and cells of a phase in a shuffled order */
    int      filter_on;  /* only run domains whose DxD window meets the box below */
    uint32_t fx0, fy0, fw, fh;
    orc_trace_rec *trace; uint64_t trace_cap, trace_n;
} orc_state;

static inline int is_pow2(uint32_t v) { return v && !(v & (v - 1)); }

static inline uint64_t word_index(const orc_state *s, uint32_t x, uint32_t y)
{
    return (uint64_t)(y >> 2) * (s->L >> 2) + (x >> 2);
}
static inline unsigned bit_index(uint32_t x, uint32_t y) { return 2u * (4u * (y & 3u) + (x & 3u)); }

static inline int get_sx(const orc_state *s, uint32_t x, uint32_t y)
{
    return (int)((s->lat[word_index(s, x, y)] >> bit_index(x, y)) & 1u);
}
static inline int get_sy(const orc_state *s, uint32_t x, uint32_t y)
{
    return (int)((s->lat[word_index(s, x, y)] >> (bit_index(x, y) + 1u)) & 1u);
}
static inline void flip_sx(orc_state *s, uint32_t x, uint32_t y)
{
    s->lat[word_index(s, x, y)] ^= 1u << bit_index(x, y);
}
static inline void flip_sy(orc_state *s, uint32_t x, uint32_t y)
{
    s->lat[word_index(s, x, y)] ^= 1u << (bit_index(x, y) + 1u);
}

/* init: 0 = flat, h(x,y) = (x+y)&1 (R5); 1 = flat shifted, h = -((x+y)&1). */
orc_state *orc_create(uint32_t L, uint64_t seed, int init, int track_heights)
{
    if (!is_pow2(L) || L < 4 || (init != 0 && init != 1)) return NULL;
    orc_state *s = (orc_state *)calloc(1, sizeof(orc_state));
    if (!s) return NULL;
    s->L = L; s->seed = seed;
    uint64_t nwords = (uint64_t)(L >> 2) * (L >> 2);
    s->lat = (uint32_t *)calloc(nwords, sizeof(uint32_t));
    if (!s->lat) { free(s); return NULL; }
    if (track_heights) {
        s->h = (int32_t *)calloc((uint64_t)L * L, sizeof(int32_t));
        if (!s->h) { free(s->lat); free(s); return NULL; }
    }
    /* build the slopes from the height definition, site by site */
    for (uint32_t y = 0; y < L; ++y)
        for (uint32_t x = 0; x < L; ++x) {
            int sgn = init == 0 ? 1 : -1;
            int hc = sgn * (int)((x + y) & 1u);
            int hw = sgn * (int)(((x + L - 1) + y) & 1u);   /* west neighbour  (x-1,y) */
            int hs = sgn * (int)((x + (y + L - 1)) & 1u);   /* south neighbour (x,y-1) */
            if (hc - hw == 1) flip_sx(s, x, y);            /* bit 1 <=> slope +1 */
            if (hc - hs == 1) flip_sy(s, x, y);
            if (s->h) s->h[(uint64_t)y * L + x] = hc;
        }
    s->h00 = 0;
    return s;
}

void orc_destroy(orc_state *s)
{
    if (!s) return;
    free(s->lat); free(s->h); free(s);
}

uint32_t *orc_lattice(orc_state *s) { return s->lat; }
int32_t  *orc_tracked_heights(orc_state *s) { return s->h; }
uint64_t  orc_mcs(const orc_state *s) { return s->t; }
int64_t   orc_net(const orc_state *s) { return s->net; }
int64_t   orc_h00(const orc_state *s) { return s->h00; }
void      orc_set_time(orc_state *s, uint64_t t) { s->t = t; }
void      orc_set_anchor(orc_state *s, int64_t h00, int64_t net) { s->h00 = h00; s->net = net; }
void      orc_set_shuffle(orc_state *s, uint64_t shuffle_seed) { s->shuffle = shuffle_seed; }
void      orc_set_filter(orc_state *s, int on, uint32_t x0, uint32_t y0, uint32_t w, uint32_t h)
{
    s->filter_on = on; s->fx0 = x0; s->fy0 = y0; s->fw = w; s->fh = h;
}
void      orc_set_trace(orc_state *s, orc_trace_rec *buf, uint64_t cap)
{
    s->trace = buf; s->trace_cap = cap; s->trace_n = 0;
}
uint64_t  orc_trace_count(const orc_state *s) { return s->trace_n; }

static void trace_push(orc_state *s, uint32_t x, uint32_t y, uint32_t set, uint32_t dom, uint32_t k,
                       uint32_t cell, int cls, int result)
{
    if (!s->trace) return;
    if (s->trace_n < s->trace_cap) {
        orc_trace_rec *r = &s->trace[s->trace_n];
        r->x = x; r->y = y; r->t = (uint32_t)s->t; r->set = set; r->dom = dom; r->k = k; r->cell = cell;
        r->cls = cls; r->result = result;
    }
    s->trace_n++;
}

/* probability -> 16-bit threshold (R18): accept iff r16 < P16. */
uint32_t orc_prob16(double p)
{
    if (!(p >= 0.0)) return 0;
    double v = p * 65536.0 + 0.5;
    if (v >= 65536.0) return 65536u;
    return (uint32_t)v;
}

/* ---------------------------------------------------------------------------------- update rule */

/* Decision of Eq. (1) at site (X,Y) on the CURRENT state: +1 deposit, -1 remove, 0 nothing.
 * b = (sx(X,Y), sx(X+1,Y), sy(X,Y), sy(X,Y+1)); local minimum (0,1,0,1) -> deposit w.p. p;
 * local maximum (1,0,1,0) -> remove w.p. q. */
static int decide(const orc_state *s, uint32_t X, uint32_t Y, uint32_t r16, uint32_t P16, uint32_t Q16)
{
    uint32_t m = s->L - 1;
    int a = get_sx(s, X, Y), b = get_sx(s, (X + 1) & m, Y);
    int c = get_sy(s, X, Y), d = get_sy(s, X, (Y + 1) & m);
    if (a == 0 && b == 1 && c == 0 && d == 1 && r16 < P16) return +1;
    if (a == 1 && b == 0 && c == 1 && d == 0 && r16 < Q16) return -1;
    return 0;
}

/* Carry out a decision: flip the four slope bits, h(X,Y) += 2*dir. */
static void apply(orc_state *s, uint32_t X, uint32_t Y, int dir)
{
    if (!dir) return;
    uint32_t m = s->L - 1;
    flip_sx(s, X, Y); flip_sx(s, (X + 1) & m, Y);
    flip_sy(s, X, Y); flip_sy(s, X, (Y + 1) & m);
    s->net += dir;
    if (X == 0 && Y == 0) s->h00 += 2 * dir;
    if (s->h) s->h[(uint64_t)Y * s->L + X] += 2 * dir;
}

/* One complete update attempt (exported for the brute-force pins). */
int orc_attempt(orc_state *s, uint32_t X, uint32_t Y, uint32_t r16, uint32_t P16, uint32_t Q16)
{
    int d = decide(s, X, Y, r16, P16, Q16);
    apply(s, X, Y, d);
    return d;
}

/* -------------------------------------------------------------------------- RS (true sequential) */

int orc_sweep_rs(orc_state *s, uint64_t n_mcs, double p, double q)
{
    uint32_t P16 = orc_prob16(p), Q16 = orc_prob16(q);
    uint32_t key[2] = { (uint32_t)s->seed, (uint32_t)(s->seed >> 32) };
    uint64_t N = (uint64_t)s->L * s->L;
    for (uint64_t i = 0; i < n_mcs; ++i) {
        for (uint64_t n = 0; n < N; ++n) {
            uint32_t ctr[4] = { (uint32_t)n, (uint32_t)(n >> 32), (uint32_t)TAG_RS << 30, (uint32_t)s->t };
            uint32_t o[4];
            orc_philox4x32_10(ctr, key, o);
            uint32_t X = o[0] & (s->L - 1), Y = o[1] & (s->L - 1), r16 = o[2] >> 16;
            int d = orc_attempt(s, X, Y, r16, P16, Q16);
            trace_push(s, X, Y, 0, 0, 0, 0, -1, d);
        }
        s->t++;
    }
    return 0;
}

/* ------------------------------------------------------------------------------- DD schemes */

/* scheme = dev | blk<<4 | tcx<<8 | tcy<<12 | log2D<<16 | ka<<21 | w<<23   (include/oct.h)
 * ka (dead-border layers only): t_async = 2^-ka MCS, i.e. 2^ka asynchronous intervals per sweep (:204-206, R27);
 * w  (dead-border layers only): dead-border width in sites, 0 = the scheme's own (DB 5, cDB 1; :166, :196-202, R22/R28). */
enum { DEV_DTR = 0, DEV_DT = 1, DEV_DB = 2, DEV_CDB = 3, DEV_DBH = 4 };
enum { BLK_DB_AUTO = 0, BLK_DB_DELAYED = 1, BLK_DT = 2, BLK_DTR = 3 };

/* tiny xorshift used ONLY by the order-shuffling test hook */
static uint64_t xs64(uint64_t *st) { uint64_t v = *st; v ^= v << 13; v ^= v >> 7; v ^= v << 17; return *st = v; }
static void shuffle_u32(uint32_t *a, uint32_t n, uint64_t *st)
{
    for (uint32_t i = n; i > 1; --i) { uint32_t j = (uint32_t)(xs64(st) % i); uint32_t tmp = a[i-1]; a[i-1] = a[j]; a[j] = tmp; }
}

typedef struct { uint32_t X, Y; uint32_t r16; int cls; int dead; } attempt_t;

/* Block-layer sweep of one device-layer domain (Sec. 3.1 :168-174): cx*cy collective single-hit
 * steps; in each step every thread cell receives exactly one attempt.  (gx,gy) = global origin of the
 * DxD domain; dead_w = device-layer dead-border width (0 for DT/DTr). */
static int domain_sweep(orc_state *s, uint32_t set, uint32_t dom, uint32_t gx, uint32_t gy,
                        uint32_t D, uint32_t cx, uint32_t cy, int blk, uint32_t dead_w,
                        uint32_t P16, uint32_t Q16, uint64_t *shuf, uint32_t k_begin, uint32_t k_end)
{
    const uint32_t key[2] = { (uint32_t)s->seed, (uint32_t)(s->seed >> 32) };
    const uint32_t ncx = D / cx, ncy = D / cy, ncell = ncx * ncy, nsteps = cx * cy, m = s->L - 1;
    const uint32_t c2c = ((uint32_t)TAG_CELL << 30) | (set << 28) | dom;
    const uint32_t c2b = ((uint32_t)TAG_BLOCK << 30) | (set << 28) | dom;
    const int delayed = (blk == BLK_DB_DELAYED) || (blk == BLK_DB_AUTO && P16 > 0 && Q16 > 0);

    uint32_t *wcache = (uint32_t *)malloc((size_t)ncell * 4 * sizeof(uint32_t)); /* memo of Philox outputs */
    attempt_t *att   = (attempt_t *)malloc((size_t)ncell * sizeof(attempt_t));
    int *dec         = (int *)malloc((size_t)ncell * sizeof(int));
    uint32_t *order  = (uint32_t *)malloc((size_t)ncell * sizeof(uint32_t));
    if (!wcache || !att || !dec || !order) { free(wcache); free(att); free(dec); free(order); return -3; }

    (void)nsteps;   /* a full sweep is k_begin = 0, k_end = cx*cy; DB with t_async = 1/2 runs half of it */
    for (uint32_t k = k_begin; k < k_end; ++k) {
        /* block-step word B for (t, set, dom, k) */
        uint32_t bo[4], bctr[4] = { k >> 2, 0, c2b, (uint32_t)s->t };
        orc_philox4x32_10(bctr, key, bo);
        const uint32_t B = bo[k & 3];

        /* attempt word w for (t, set, dom, cell, k): one Philox call serves 4 consecutive steps */
        if ((k & 3) == 0 || k == k_begin)
            for (uint32_t c = 0; c < ncell; ++c) {
                uint32_t cctr[4] = { k >> 2, c, c2c, (uint32_t)s->t };
                orc_philox4x32_10(cctr, key, &wcache[4 * c]);
            }

        for (uint32_t c = 0; c < ncell; ++c) {
            const uint32_t a = c % ncx, b = c / ncx, w = wcache[4 * c + (k & 3)];
            uint32_t x, y; int cls;
            if (blk == BLK_DT || blk == BLK_DTR) {     /* :170, random quadrant per step */
                const uint32_t Q = (B >> 16) & 3u;
                const uint32_t lx = w & (cx / 2 - 1), ly = (w >> 8) & (cy / 2 - 1);
                x = a * cx + (Q & 1u) * (cx / 2) + lx;
                y = b * cy + (Q >> 1) * (cy / 2) + ly;
                if (blk == BLK_DTR) {                  /* :234 "DTrDTr": the block-layer origin also moves
                                                          after each collective update (R26): the
                                                          same origin draw as block-layer DB, cells wrap (R14) */
                    x = (x + (B & (cx - 1))) & (D - 1);
                    y = (y + ((B >> 8) & (cy - 1))) & (D - 1);
                }
                cls = -1;
            } else {                                   /* :172, DB with random origin per step */
                const uint32_t ox = B & (cx - 1), oy = (B >> 8) & (cy - 1);
                const uint32_t lx = w & (cx - 1), ly = (w >> 8) & (cy - 1);
                x = (a * cx + lx + ox) & (D - 1);
                y = (b * cy + ly + oy) & (D - 1);
                cls = (lx == cx - 1) + (ly == cy - 1);
            }
            att[c].X = (gx + x) & m; att[c].Y = (gy + y) & m;
            att[c].r16 = w >> 16; att[c].cls = cls;
            att[c].dead = dead_w && (x >= D - dead_w || y >= D - dead_w);   /* :135 */
            order[c] = c;
        }
        if (shuf) shuffle_u32(order, ncell, shuf);

        if (blk == BLK_DT || blk == BLK_DTR) {
            for (uint32_t i = 0; i < ncell; ++i) {
                const attempt_t *A = &att[order[i]];
                int d = A->dead ? 0 : orc_attempt(s, A->X, A->Y, A->r16, P16, Q16);
                trace_push(s, A->X, A->Y, set, dom, k, order[i], -1, A->dead ? 2 : d);
            }
        } else if (!delayed) {
            /* "ignoring borders" (:174), made order-free: decide all on the step's initial state,
             * then apply all (R16) */
            for (uint32_t i = 0; i < ncell; ++i) {
                const attempt_t *A = &att[order[i]];
                dec[order[i]] = A->dead ? 0 : decide(s, A->X, A->Y, A->r16, P16, Q16);
            }
            if (shuf) shuffle_u32(order, ncell, shuf);
            for (uint32_t i = 0; i < ncell; ++i) {
                const attempt_t *A = &att[order[i]];
                apply(s, A->X, A->Y, dec[order[i]]);
                trace_push(s, A->X, A->Y, set, dom, k, order[i], A->cls, A->dead ? 2 : dec[order[i]]);
            }
        } else {
            /* delayed borders (:174): bulk, then edges, then corners */
            for (int phase = 0; phase < 3; ++phase) {
                for (uint32_t i = 0; i < ncell; ++i) {
                    const attempt_t *A = &att[order[i]];
                    if (A->cls != phase) continue;
                    int d = A->dead ? 0 : orc_attempt(s, A->X, A->Y, A->r16, P16, Q16);
                    trace_push(s, A->X, A->Y, set, dom, k, order[i], A->cls, A->dead ? 2 : d);
                }
            }
        }
    }
    free(wcache); free(att); free(dec); free(order);
    return 0;
}

/* periodic interval test: does [a, a+la) meet [b, b+lb) on a ring of length L? */
static int ring_meets(uint32_t a, uint32_t la, uint32_t b, uint32_t lb, uint32_t L)
{
    return ((a - b) & (L - 1)) < lb || ((b - a) & (L - 1)) < la;
}

/* the idx-th permutation of (0,1,2,3) in lexicographic order (factorial number system) */
static void lex_perm4(uint32_t idx, uint32_t perm[4])
{
    uint32_t pool[4] = { 0, 1, 2, 3 }, n = 4, f = 6;   /* 3! */
    for (uint32_t i = 0; i < 4; ++i) {
        uint32_t j = idx / f; idx %= f;
        perm[i] = pool[j];
        for (uint32_t r = j; r + 1 < n; ++r) pool[r] = pool[r + 1];
        --n;
        if (n > 1) f /= (n);   /* 6 -> 2 -> 1 */
    }
}

int orc_check_scheme(uint32_t L, uint32_t scheme)
{
    const uint32_t dev = scheme & 15u, blk = (scheme >> 4) & 15u, tcx = (scheme >> 8) & 15u,
                   tcy = (scheme >> 12) & 15u, lD = (scheme >> 16) & 31u, ka = (scheme >> 21) & 3u, w = (scheme >> 23) & 7u;
    if ((scheme >> 26) != 0 || dev > 4 || blk > 3 || lD < 3 || lD > 12) return -1;
    if ((ka || w) && dev != DEV_DB && dev != DEV_CDB) return -1;   /* t_async and width belong to the dead-border layers; DBh is DB with ka = 1 */
    if (ka > 2) return -1;                                          /* the interval index shares the 2-bit set field of the counters (R19) */
    const uint32_t D = 1u << lD, cx = 4u << tcx, cy = 4u << tcy;
    if (w >= D || ((cx * cy) >> ka) < 4 || ((cx * cy) >> ka) % 4 != 0) return -1;   /* whole Philox calls (4 steps) per interval */
    if (cx > 64 || cy > 64 || cx > D || cy > D) return -1;
    if ((blk == BLK_DT || blk == BLK_DTR) && (tcx < 1 || tcy < 1)) return -1;   /* :182 smallest TC=1,1 for DT */
    if (!is_pow2(L)) return -1;
    if ((dev == DEV_DTR || dev == DEV_DT) ? (L < 2 * D) : (L < D)) return -1;
    const uint64_t ntile = (dev <= DEV_DT) ? (uint64_t)(L / (2 * D)) * (L / (2 * D)) : (uint64_t)(L / D) * (L / D);
    if (ntile > (1u << 28)) return -1;
    return 0;
}

int orc_sweep_dd(orc_state *s, uint64_t n_mcs, double p, double q, uint32_t scheme)
{
    if (orc_check_scheme(s->L, scheme)) return -1;
    const uint32_t dev = scheme & 15u, blk = (scheme >> 4) & 15u, tcx = (scheme >> 8) & 15u,
                   tcy = (scheme >> 12) & 15u, lD = (scheme >> 16) & 31u, ka = (scheme >> 21) & 3u, wsel = (scheme >> 23) & 7u;
    const uint32_t D = 1u << lD, cx = 4u << tcx, cy = 4u << tcy, L = s->L, m = L - 1;
    const uint32_t P16 = orc_prob16(p), Q16 = orc_prob16(q);
    const uint32_t key[2] = { (uint32_t)s->seed, (uint32_t)(s->seed >> 32) };
    uint64_t shuf_state = s->shuffle, *shuf = s->shuffle ? &shuf_state : NULL;

    for (uint64_t i = 0; i < n_mcs; ++i) {
        if (s->t > 0xFFFFFFFFull) return -1;
        uint32_t G[4], gctr[4] = { 0, 0, (uint32_t)TAG_GLOBAL << 30, (uint32_t)s->t };
        orc_philox4x32_10(gctr, key, G);

        if (dev == DEV_DTR || dev == DEV_DT) {
            /* :144 four domain sets in a freshly shuffled permutation; :150 random origin (DTr) */
            const uint32_t Ox = dev == DEV_DTR ? (G[0] & m) : 0, Oy = dev == DEV_DTR ? (G[1] & m) : 0;
            uint32_t perm[4];
            lex_perm4(G[2] % 24u, perm);
            const uint32_t nt = L / (2 * D);
            uint32_t *dorder = (uint32_t *)malloc((size_t)nt * nt * sizeof(uint32_t));
            if (!dorder) return -3;
            for (uint32_t si = 0; si < 4; ++si) {
                const uint32_t set = perm[si], sx = set & 1u, sy = set >> 1;
                for (uint32_t d = 0; d < nt * nt; ++d) dorder[d] = d;
                if (shuf) shuffle_u32(dorder, nt * nt, shuf);
                for (uint32_t di = 0; di < nt * nt; ++di) {
                    const uint32_t dom = dorder[di], I = dom % nt, J = dom / nt;
                    const uint32_t gx = (Ox + 2 * D * I + sx * D) & m, gy = (Oy + 2 * D * J + sy * D) & m;
                    if (s->filter_on && !(ring_meets(gx, D, s->fx0, s->fw, L) && ring_meets(gy, D, s->fy0, s->fh, L)))
                        continue;
                    int rc = domain_sweep(s, set, dom, gx, gy, D, cx, cy, (int)blk, 0, P16, Q16, shuf, 0, cx * cy);
                    if (rc) { free(dorder); return rc; }
                }
            }
            free(dorder);
        } else {
            /* :135 dead border; :166 cDB = origin on the 4x4 word grid, border 1; DB = free origin, border 5.
             * t_async = 1/n_int MCS (:204-206, R27; DBh = DB with two intervals): n_int intervals per sweep, each
             * with its own origin (global stream c0 = interval) and 1/n_int of the collective steps. */
            const uint32_t n_int = dev == DEV_DBH ? 2u : (1u << ka);              /* t_async = 1 / n_int MCS (:204-206) */
            const uint32_t dead_w = wsel ? wsel : (dev == DEV_CDB ? 1u : 5u);     /* :166; explicit width: :202, R28 */
            const uint32_t nt = L / D;
            uint32_t *dorder = (uint32_t *)malloc((size_t)nt * nt * sizeof(uint32_t));
            if (!dorder) return -3;
            for (uint32_t iv = 0; iv < n_int; ++iv) {
                if (iv > 0) { gctr[0] = iv; orc_philox4x32_10(gctr, key, G); }
                const uint32_t Ox = dev == DEV_CDB ? (G[0] & m & ~3u) : (G[0] & m);
                const uint32_t Oy = dev == DEV_CDB ? (G[1] & m & ~3u) : (G[1] & m);
                const uint32_t k_begin = iv * (cx * cy / n_int), k_end = (iv + 1) * (cx * cy / n_int);
                for (uint32_t d = 0; d < nt * nt; ++d) dorder[d] = d;
                if (shuf) shuffle_u32(dorder, nt * nt, shuf);
                for (uint32_t di = 0; di < nt * nt; ++di) {
                    const uint32_t dom = dorder[di], I = dom % nt, J = dom / nt;
                    const uint32_t gx = (Ox + D * I) & m, gy = (Oy + D * J) & m;
                    if (s->filter_on && !(ring_meets(gx, D, s->fx0, s->fw, L) && ring_meets(gy, D, s->fy0, s->fh, L)))
                        continue;
                    int rc = domain_sweep(s, iv, dom, gx, gy, D, cx, cy, (int)blk, dead_w, P16, Q16, shuf, k_begin, k_end);
                    if (rc) { free(dorder); return rc; }
                }
            }
            free(dorder);
        }
        s->t++;
    }
    return 0;
}

/* Per-MCS control values alone (R10/R19), exported so tests can pin them. */
void orc_mcs_control(uint64_t seed, uint32_t t, uint32_t L, uint32_t dev, uint32_t out[6])
{
    const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t G[4], gctr[4] = { 0, 0, (uint32_t)TAG_GLOBAL << 30, t }, perm[4];
    orc_philox4x32_10(gctr, key, G);
    lex_perm4(G[2] % 24u, perm);
    uint32_t Ox = G[0] & (L - 1), Oy = G[1] & (L - 1);
    if (dev == DEV_DT) { Ox = 0; Oy = 0; }
    if (dev == DEV_CDB) { Ox &= ~3u; Oy &= ~3u; }
    out[0] = Ox; out[1] = Oy; out[2] = perm[0]; out[3] = perm[1]; out[4] = perm[2]; out[5] = perm[3];
}

/* ------------------------------------------------------------------------- heights & observables */

/* h(x,0) = h00 + sum_{i=1..x} sx(i,0);  h(x,y) = h(x,0) + sum_{j=1..y} sy(x,j)   (:52; R20) */
void orc_heights(const orc_state *s, int32_t *out)
{
    const uint32_t L = s->L;
    for (uint32_t x = 0; x < L; ++x) {
        int32_t h = (int32_t)s->h00;
        for (uint32_t i = 1; i <= x; ++i) h += get_sx(s, i, 0) ? 1 : -1;
        out[x] = h;
        for (uint32_t y = 1; y < L; ++y) {
            h += get_sy(s, x, y) ? 1 : -1;
            out[(uint64_t)y * L + x] = h;
        }
    }
}

/* the other path: first up column 0, then along each row */
void orc_heights_rowpath(const orc_state *s, int32_t *out)
{
    const uint32_t L = s->L;
    for (uint32_t y = 0; y < L; ++y) {
        int32_t h = (int32_t)s->h00;
        for (uint32_t j = 1; j <= y; ++j) h += get_sy(s, 0, j) ? 1 : -1;
        out[(uint64_t)y * L] = h;
        for (uint32_t x = 1; x < L; ++x) {
            h += get_sx(s, x, y) ? 1 : -1;
            out[(uint64_t)y * L + x] = h;
        }
    }
}

/* out = {S1 = sum(h-c), S2 = sum (h-c)^2, c = h(0,0), net}; W^2 = S2/N - (S1/N)^2  (Eq. (3) :61) */
int orc_sums(const orc_state *s, int64_t out[4])
{
    const uint64_t N = (uint64_t)s->L * s->L;
    int32_t *h = (int32_t *)malloc(N * sizeof(int32_t));
    if (!h) return -3;
    orc_heights(s, h);
    int64_t S1 = 0, S2 = 0, c = s->h00;
    for (uint64_t i = 0; i < N; ++i) { int64_t d = (int64_t)h[i] - c; S1 += d; S2 += d * d; }
    free(h);
    out[0] = S1; out[1] = S2; out[2] = c; out[3] = s->net;
    return 0;
}

/* The same four numbers as orc_sums along the OTHER integration path (up column 0, then along each row, as in
 * orc_heights_rowpath) without materialising the heights: O(1) extra memory, so it also serves L = 2^17, where the
 * int32 height array would take 64 GiB.  Pinned against orc_sums (tests/test_oracle_rule.py). */
int orc_sums_rowpath(const orc_state *s, int64_t out[4])
{
    const uint32_t L = s->L;
    int64_t S1 = 0, S2 = 0, col = 0;                    /* col = h(0,y) - c */
    for (uint32_t y = 0; y < L; ++y) {
        if (y > 0) col += get_sy(s, 0, y) ? 1 : -1;
        int64_t d = col;
        S1 += d; S2 += d * d;
        for (uint32_t x = 1; x < L; ++x) {
            d += get_sx(s, x, y) ? 1 : -1;
            S1 += d; S2 += d * d;
        }
    }
    out[0] = S1; out[1] = S2; out[2] = s->h00; out[3] = s->net;
    return 0;
}

/* out = {S_t, S_s, S_ts, c_t, c_s}: C_h(t,s) = S_ts/N - (S_t/N)(S_s/N)   (Eq. (6) :92, reading R7) */
int orc_autocorr_sums(const orc_state *now, const orc_state *snap, int64_t out[5])
{
    if (now->L != snap->L) return -1;
    const uint64_t N = (uint64_t)now->L * now->L;
    int32_t *ht = (int32_t *)malloc(N * sizeof(int32_t)), *hs = (int32_t *)malloc(N * sizeof(int32_t));
    if (!ht || !hs) { free(ht); free(hs); return -3; }
    orc_heights(now, ht); orc_heights(snap, hs);
    int64_t St = 0, Ss = 0, Sts = 0, ct = now->h00, cs = snap->h00;
    for (uint64_t i = 0; i < N; ++i) {
        int64_t a = (int64_t)ht[i] - ct, b = (int64_t)hs[i] - cs;
        St += a; Ss += b; Sts += a * b;
    }
    free(ht); free(hs);
    out[0] = St; out[1] = Ss; out[2] = Sts; out[3] = ct; out[4] = cs;
    return 0;
}

/* Slope autocorrelation (:85-88): C_s(t,s) = <n(t,r) n(s,r)> - <n(t)><n(s)> with n the lattice-gas
 * occupation = the slope bit (:50 "up/down slopes ... particles/holes").  Integer sums, x and y slopes
 * kept apart: out = {sum nx_t nx_s, sum ny_t ny_s, sum nx_t, sum ny_t, sum nx_s, sum ny_s}. */
int orc_slope_autocorr_sums(const orc_state *now, const orc_state *snap, int64_t out[6])
{
    if (now->L != snap->L) return -1;
    const uint32_t L = now->L;
    for (int k = 0; k < 6; ++k) out[k] = 0;
    for (uint32_t y = 0; y < L; ++y)
        for (uint32_t x = 0; x < L; ++x) {
            const int xt = get_sx(now, x, y), yt = get_sy(now, x, y);
            const int xs = get_sx(snap, x, y), ys = get_sy(snap, x, y);
            out[0] += xt * xs; out[1] += yt * ys;
            out[2] += xt; out[3] += yt; out[4] += xs; out[5] += ys;
        }
    return 0;
}

/* a copy of the state (waiting-time snapshot for aging, :80) */
orc_state *orc_clone(const orc_state *s)
{
    orc_state *c = (orc_state *)calloc(1, sizeof(orc_state));
    if (!c) return NULL;
    *c = *s; c->trace = NULL; c->trace_cap = c->trace_n = 0;
    uint64_t nwords = (uint64_t)(s->L >> 2) * (s->L >> 2);
    c->lat = (uint32_t *)malloc(nwords * sizeof(uint32_t));
    if (!c->lat) { free(c); return NULL; }
    memcpy(c->lat, s->lat, nwords * sizeof(uint32_t));
    c->h = NULL;
    if (s->h) {
        c->h = (int32_t *)malloc((uint64_t)s->L * s->L * sizeof(int32_t));
        if (!c->h) { free(c->lat); free(c); return NULL; }
        memcpy(c->h, s->h, (uint64_t)s->L * s->L * sizeof(int32_t));
    }
    return c;
}

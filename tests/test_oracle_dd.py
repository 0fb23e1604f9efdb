"""Pins for the oracle's domain-decomposition loops (Sec. 3, :129-182; DESIGN.md readings).

The attempt trace is checked against what the paper fixes: 1 MCS = L^2 attempts (:106); four
non-interacting domain sets that are visited in a shuffled permutation (:144); every thread cell
receives exactly one attempt per collective step (:168); DB cells are the aligned cells displaced by
one common random origin and wrap inside the domain (:172, R14); DT picks one quadrant per step (:170);
dead-border hits are not carried out (:135).  Order independence, split invariance and the
deposition/removal symmetry pin the loop nest against dropped or transposed indices.
"""
import itertools

import numpy as np
import pytest

import oracle
from oracle import BLK_DB, BLK_DB_DELAYED, BLK_DT, BLK_DTR, DEV_CDB, DEV_DB, DEV_DBH, DEV_DT, DEV_DTR, Oracle, scheme


def run_traced(L, seed, code, n_mcs, p=1.0, q=0.0, t0=0):
    o = Oracle(L, seed)
    if t0:
        o.set_lattice(o.lattice.copy(), t=t0)
    o.start_trace(n_mcs * L * L + 16)
    o.sweep(n_mcs, p, q, code)
    tr = o.stop_trace()
    return o, tr


def dims(code):
    return 1 << ((code >> 16) & 31), 4 << ((code >> 8) & 15), 4 << ((code >> 12) & 15)


@pytest.mark.parametrize("code", [scheme(DEV_DTR, BLK_DB, 5), scheme(DEV_DTR, BLK_DB, 5, 2, 1),
                                  scheme(DEV_DT, BLK_DB_DELAYED, 5), scheme(DEV_DTR, BLK_DB, 4, 0, 0)])
def test_dtr_db_trace_geometry(code):
    L, seed = 128, 21
    D, cx, cy = dims(code)
    dev = code & 15
    o, tr = run_traced(L, seed, code, 2, p=0.6, q=0.4 if (code >> 4) & 15 == BLK_DB_DELAYED else 0.0)
    assert len(tr) == 2 * L * L                                        # :106
    nt = L // (2 * D)
    for t in (0, 1):
        Ox, Oy, perm = oracle.mcs_control(seed, t, L, dev)
        if dev == DEV_DT:
            assert (Ox, Oy) == (0, 0)
        rec = tr[tr["t"] == t]
        # sets appear in the order of the permutation, each one complete before the next (:144)
        set_seq = [k for k, _ in itertools.groupby(rec["set"].tolist())]
        assert tuple(set_seq) == perm and sorted(perm) == [0, 1, 2, 3]
        cover = np.zeros((L, L), dtype=np.int32)
        for s in range(4):
            rs = rec[rec["set"] == s]
            assert len(rs) == L * L // 4
            assert set(rs["dom"].tolist()) == set(range(nt * nt))
            for dom in range(nt * nt):
                rd = rs[rs["dom"] == dom]
                assert len(rd) == D * D                                # one sweep of the domain (R12)
                I, J = dom % nt, dom // nt
                gx = (Ox + 2 * D * I + (s & 1) * D) % L
                gy = (Oy + 2 * D * J + (s >> 1) * D) % L
                lx = (rd["x"].astype(np.int64) - gx) % L
                ly = (rd["y"].astype(np.int64) - gy) % L
                assert (lx < D).all() and (ly < D).all()               # inside its own sub-tile
                cover[gy:gy + 1, gx:gx + 1] += 0
                yy = (gy + np.arange(D)) % L
                xx = (gx + np.arange(D)) % L
                cover[np.ix_(yy, xx)] += 1
                ncx = D // cx
                for k in range(cx * cy):
                    rk = rd[rd["k"] == k]
                    assert sorted(rk["cell"].tolist()) == list(range((D // cx) * (D // cy)))   # single hit (:168)
                    a, b = rk["cell"] % ncx, rk["cell"] // ncx
                    klx, kly = (rk["x"].astype(np.int64) - gx) % L, (rk["y"].astype(np.int64) - gy) % L
                    # one common origin (ox,oy) per step explains every cell's site (:172, R13/R14)
                    ok = [(ox, oy) for ox in range(cx) for oy in range(cy)
                          if ((((klx - ox) % D) // cx) == a).all() and ((((kly - oy) % D) // cy) == b).all()]
                    assert len(ok) >= 1
                    ox, oy = ok[0]
                    inx, iny = (klx - ox) % D - a * cx, (kly - oy) % D - b * cy
                    cls = (inx == cx - 1).astype(int) + (iny == cy - 1).astype(int)
                    if len(ok) == 1:
                        assert (cls == rk["cls"]).all()                # +x column / +y row are the border (R15)
        assert (cover == 1).all()                                      # the 4 sets tile the lattice exactly
    o.close()


def test_delayed_phases_are_ordered_bulk_edges_corners():
    code = scheme(DEV_DTR, BLK_DB_DELAYED, 5)
    o, tr = run_traced(64, 4, code, 1, p=0.5, q=0.5)
    for (s, d, k), grp in itertools.groupby(tr, key=lambda r: (r["set"], r["dom"], r["k"])):
        cls = [int(r["cls"]) for r in grp]
        assert cls == sorted(cls)                                      # :174 "corners ... last"
    o.close()


@pytest.mark.parametrize("code", [scheme(DEV_DTR, BLK_DT, 5), scheme(DEV_DTR, BLK_DT, 5, 2, 1)])
def test_dt_block_layer_trace(code):
    L, seed = 64, 8
    D, cx, cy = dims(code)
    o, tr = run_traced(L, seed, code, 2)
    assert len(tr) == 2 * L * L
    quads = []
    for t in (0, 1):
        Ox, Oy, perm = oracle.mcs_control(seed, t, L, DEV_DTR)
        rec = tr[tr["t"] == t]
        nt = L // (2 * D)
        for s in range(4):
            for dom in range(nt * nt):
                rd = rec[(rec["set"] == s) & (rec["dom"] == dom)]
                gx = (Ox + 2 * D * (dom % nt) + (s & 1) * D) % L
                gy = (Oy + 2 * D * (dom // nt) + (s >> 1) * D) % L
                lx, ly = (rd["x"].astype(np.int64) - gx) % L, (rd["y"].astype(np.int64) - gy) % L
                assert (lx < D).all() and (ly < D).all()
                a, b = rd["cell"] % (D // cx), rd["cell"] // (D // cx)
                assert ((lx // cx) == a).all() and ((ly // cy) == b).all()     # aligned cells, no wrap
                qx, qy = (lx % cx) // (cx // 2), (ly % cy) // (cy // 2)
                for k in range(cx * cy):
                    m = rd["k"] == k
                    assert m.sum() == (D // cx) * (D // cy)
                    assert len(set(qx[m].tolist())) == 1 and len(set(qy[m].tolist())) == 1   # one quadrant per step (R17)
                    quads.append(int(qx[m][0]) + 2 * int(qy[m][0]))
    # drawn with replacement, all four occur, roughly uniformly (:170 "at random", not a permutation)
    cnt = np.bincount(quads, minlength=4)
    assert (cnt > 0.15 * len(quads)).all()
    runs = sum(1 for i in range(0, len(quads) - 3, 4) if sorted(quads[i:i + 4]) == [0, 1, 2, 3])
    assert runs < 0.5 * (len(quads) // 4)
    o.close()


@pytest.mark.parametrize("code", [scheme(DEV_DTR, BLK_DTR, 5), scheme(DEV_DTR, BLK_DTR, 5, 2, 1)])
def test_dtr_block_layer_trace(code):
    """Block-layer DTr ("DTrDTr", R26): block-layer DT whose origin moves after each collective
    update.  Per step all cells select inside one common quadrant (as DT) of their cell displaced by one
    common origin (as DB) with wrap inside the domain; every cell is hit once per step, the origins are
    uniform on [0,cx) x [0,cy), and with origin (0,0) the selection is exactly DT's."""
    L, seed = 64, 9
    D, cx, cy = dims(code)
    o, tr = run_traced(L, seed, code, 2)
    assert len(tr) == 2 * L * L
    origins = []
    for t in (0, 1):
        Ox, Oy, perm = oracle.mcs_control(seed, t, L, DEV_DTR)
        rec = tr[tr["t"] == t]
        nt = L // (2 * D)
        for s in range(4):
            for dom in range(nt * nt):
                rd = rec[(rec["set"] == s) & (rec["dom"] == dom)]
                gx = (Ox + 2 * D * (dom % nt) + (s & 1) * D) % L
                gy = (Oy + 2 * D * (dom // nt) + (s >> 1) * D) % L
                lx, ly = (rd["x"].astype(np.int64) - gx) % L, (rd["y"].astype(np.int64) - gy) % L
                assert (lx < D).all() and (ly < D).all()
                a, b = rd["cell"] % (D // cx), rd["cell"] // (D // cx)
                for k in range(cx * cy):
                    m = rd["k"] == k
                    assert m.sum() == (D // cx) * (D // cy) and len(set(rd["cell"][m].tolist())) == m.sum()
                    # offsets from the cells' own corners, modulo the domain: all inside ONE window of
                    # (cx/2) x (cy/2) sites = quadrant corner + common origin
                    ux, uy = (lx[m] - a[m] * cx) % D, (ly[m] - b[m] * cy) % D
                    for u, half, full in ((ux, cx // 2, cx), (uy, cy // 2, cy)):
                        starts = [s0 for s0 in range(0, 2 * full) if all(((int(v) - s0) % D) < half for v in u)]
                        assert starts, "cells of one step do not share a quadrant window"
                    origins.append((int(ux.min()), int(uy.min())))
    # the windows start anywhere in [0, cx + cx/2): quadrant offset {0, cx/2} + origin [0, cx)
    xs = np.array([v[0] for v in origins]); ys = np.array([v[1] for v in origins])
    assert xs.max() >= cx and ys.max() >= cy // 2 and xs.min() < 4 and ys.min() < 4
    # against plain DT: identical attempts whenever the drawn origin is (0,0); different otherwise
    o_dt, tr_dt = run_traced(L, seed, (code & ~0xF0) | (BLK_DT << 4), 2)
    same = (tr["x"] == tr_dt["x"]) & (tr["y"] == tr_dt["y"])
    assert 0 < same.mean() < 0.2
    o.close(); o_dt.close()


@pytest.mark.parametrize("dev,w", [(DEV_DB, 5), (DEV_CDB, 1)])
def test_dead_border_device_layer(dev, w):
    L, seed, code = 128, 17, scheme(dev, BLK_DB, 5)
    D = 32
    o, tr = run_traced(L, seed, code, 3)
    assert len(tr) == 3 * L * L
    for t in range(3):
        Ox, Oy, _ = oracle.mcs_control(seed, t, L, dev)
        if dev == DEV_CDB:
            assert Ox % 4 == 0 and Oy % 4 == 0                        # :166 coarse grid
        rec = tr[tr["t"] == t]
        lx = (rec["x"].astype(np.int64) - Ox) % D
        ly = (rec["y"].astype(np.int64) - Oy) % D
        border = (lx >= D - w) | (ly >= D - w)
        assert ((rec["result"] == 2) == border).all()                 # border hits are not carried out (:135)
        nt = L // D
        dom = ((rec["y"].astype(np.int64) - Oy) % L) // D * nt + ((rec["x"].astype(np.int64) - Ox) % L) // D
        assert (dom == rec["dom"]).all()
        # Eq. (9), reading R9: the active fraction of a sweep
        assert abs(border.mean() - (1 - ((D - w) / D) ** 2)) < 0.01
    o.close()


def test_dead_border_half_sweep_intervals():
    """DB with t_async = 1/2 MCS (R27): a sweep is two asynchronous intervals, each with its
    own tiling origin and half of the collective steps, so every tile gets D^2/2 attempts per interval."""
    L, seed, D, cx, cy, w = 128, 23, 32, 8, 8, 5
    code = scheme(DEV_DBH, BLK_DB, 5)
    o, tr = run_traced(L, seed, code, 2)
    assert len(tr) == 2 * L * L                                       # still L^2 attempts per sweep (:106)
    nt = L // D
    moved = 0
    for t in range(2):
        rec = tr[tr["t"] == t]
        halves = (rec[rec["k"] < cx * cy // 2], rec[rec["k"] >= cx * cy // 2])
        assert len(halves[0]) == len(halves[1]) == L * L // 2
        assert (halves[0]["set"] == 0).all() and (halves[1]["set"] == 1).all()      # the interval index keys the streams
        origins = []
        for iv, part in enumerate(halves):
            # recover the interval's origin from any attempt of tile 0 / cell 0: x = O + (lx + ox) mod D ...
            # simpler and stricter: there must be ONE origin (Ox, Oy) that puts every attempt of tile `dom`
            # into that tile and every discarded attempt into the 5-wide border
            cand = None
            r0 = part[0]
            for Ox in range(L):
                if ((int(r0["x"]) - Ox) % L) // D == int(r0["dom"]) % nt:
                    lx = (part["x"].astype(np.int64) - Ox) % L
                    if ((lx // D) == part["dom"] % nt).all():
                        bx = (lx % D) >= D - w
                        cand = (Ox, bx) if cand is None else cand
                        break
            assert cand is not None
            Ox, bx = cand
            for Oy in range(L):
                ly = (part["y"].astype(np.int64) - Oy) % L
                if ((ly // D) == part["dom"] // nt).all():
                    by = (ly % D) >= D - w
                    break
            else:
                raise AssertionError("no y origin fits")
            assert ((part["result"] == 2) == (bx | by)).all()
            origins.append((Ox, Oy))
            for dom in (0, nt * nt - 1):
                assert (part["dom"] == dom).sum() == D * D // 2
        Ox0, Oy0, _ = oracle.mcs_control(seed, t, L, DEV_DB)
        assert origins[0] == (Ox0, Oy0)                                  # interval 0 = the plain DB draw (c0 = 0)
        moved += origins[0] != origins[1]
    assert moved == 2                                                     # the origin moves between the intervals
    # the first interval of DBh is exactly the first half of a DB sweep
    o_db, tr_db = run_traced(L, seed, scheme(DEV_DB, BLK_DB, 5), 1)
    first = tr[(tr["t"] == 0) & (tr["k"] < cx * cy // 2)]
    ref = tr_db[tr_db["k"] < cx * cy // 2]
    # the oracle visits tile by tile, so compare as sets of (dom, cell, k, x, y)
    key = lambda a: sorted(zip(a["dom"].tolist(), a["cell"].tolist(), a["k"].tolist(), a["x"].tolist(), a["y"].tolist()))
    assert key(first) == key(ref)
    o.close(); o_db.close()


def _fit_origin(part, L, D, nt):
    """the ONE tiling origin (Ox, Oy) that puts every traced attempt of tile `dom` into that tile"""
    found = []
    for axis, col in (("x", lambda d: d % nt), ("y", lambda d: d // nt)):
        for O in range(L):
            l = (part[axis].astype(np.int64) - O) % L
            if ((l // D) == col(part["dom"])).all():
                found.append(O)
                break
        else:
            raise AssertionError(f"no {axis} origin fits")
    return tuple(found)


@pytest.mark.parametrize("dev,ka,w", [(DEV_DB, 2, 0), (DEV_DB, 1, 0), (DEV_DB, 0, 1), (DEV_DB, 2, 1), (DEV_DB, 1, 3), (DEV_CDB, 1, 0), (DEV_CDB, 0, 2)])
def test_general_t_async_and_border_width(dev, ka, w):
    """DB / cDB with t_async = 2^-ka MCS and an explicit border width (R27/R28), from the attempt trace:
    2^ka intervals per sweep, each with its own origin (free for DB, on the 4-site grid for cDB) and 1/2^ka of the
    collective steps; an attempt is discarded iff it falls into the rim of the stated width; L^2 attempts per sweep."""
    L, seed, D, cx, cy = 128, 31, 32, 8, 8
    width = w if w else (1 if dev == DEV_CDB else 5)
    n_int = 1 << ka
    code = scheme(dev, BLK_DB, 5, 1, 1, ka, w)
    o, tr = run_traced(L, seed, code, 2, 0.8, 0.2)
    assert len(tr) == 2 * L * L
    nt, per = L // D, cx * cy // n_int
    seen = set()
    for t in range(2):
        rec = tr[tr["t"] == t]
        for iv in range(n_int):
            part = rec[(rec["k"] >= iv * per) & (rec["k"] < (iv + 1) * per)]
            assert len(part) == L * L // n_int and (part["set"] == iv).all()
            Ox, Oy = _fit_origin(part, L, D, nt)
            if dev == DEV_CDB:
                assert Ox % 4 == 0 and Oy % 4 == 0
            seen.add((Ox % 4, Oy % 4))
            lx, ly = (part["x"].astype(np.int64) - Ox) % L % D, (part["y"].astype(np.int64) - Oy) % L % D
            assert ((part["result"] == 2) == ((lx >= D - width) | (ly >= D - width))).all()
            for dom in (0, nt * nt - 1):
                assert (part["dom"] == dom).sum() == D * D // n_int
            if iv == 0:
                assert (Ox, Oy) == oracle.mcs_control(seed, t, L, dev)[:2]              # interval 0 = the plain draw (c0 = 0)
    if dev == DEV_DB and n_int * 2 >= 4:
        assert len(seen) > 1                                                            # free origin: not on a coarse grid
    # discarded fraction = border fraction N_border / N of Eq. (9)
    frac = (tr["result"] == 2).mean()
    assert abs(frac - (1 - ((D - width) / D) ** 2)) < 0.01
    o.close()


def test_t_async_and_width_reduce_to_the_named_schemes():
    L, seed = 128, 5
    runs = {}
    for name, code in (("DBh", scheme(DEV_DBH, BLK_DB, 5)), ("DB ka=1", scheme(DEV_DB, BLK_DB, 5, 1, 1, 1, 0)),
                       ("DB", scheme(DEV_DB, BLK_DB, 5)), ("DB w=5", scheme(DEV_DB, BLK_DB, 5, 1, 1, 0, 5)),
                       ("cDB", scheme(DEV_CDB, BLK_DT, 5)), ("cDB w=1", scheme(DEV_CDB, BLK_DT, 5, 1, 1, 0, 1)),
                       ("DB w=1", scheme(DEV_DB, BLK_DB, 5, 1, 1, 0, 1)), ("DB ka=2", scheme(DEV_DB, BLK_DB, 5, 1, 1, 2, 0))):
        o = Oracle(L, seed)
        o.sweep(6, 0.7, 0.3, code)
        runs[name] = (o.lattice.copy(), o.net, o.h00)
        o.close()
    same = lambda a, b: (runs[a][0] == runs[b][0]).all() and runs[a][1:] == runs[b][1:]     # noqa: E731
    assert same("DBh", "DB ka=1") and same("DB", "DB w=5") and same("cDB", "cDB w=1")
    assert not same("DB", "DB w=1") and not same("DB", "DB ka=2") and not same("DB ka=1", "DB ka=2")
    # the fields belong to the dead-border layers only; at most four intervals; whole Philox calls per interval
    chk = oracle.lib().orc_check_scheme
    assert chk(L, scheme(DEV_DTR, BLK_DB, 5, 1, 1, 1, 0)) != 0 and chk(L, scheme(DEV_DT, BLK_DB, 5, 1, 1, 0, 1)) != 0
    assert chk(L, scheme(DEV_DBH, BLK_DB, 5, 1, 1, 1, 0)) != 0 and chk(L, scheme(DEV_DB, BLK_DB, 5, 1, 1, 3, 0)) != 0
    assert chk(L, scheme(DEV_DB, BLK_DB, 5, 0, 0, 2, 0)) == 0 and chk(L, scheme(DEV_DB, BLK_DB, 5, 1, 1, 2, 7)) == 0


def test_origin_and_permutation_statistics():
    L = 1024
    ox, oy, perms = [], [], []
    for t in range(4800):
        a, b, p = oracle.mcs_control(99, t, L, DEV_DTR)
        ox.append(a); oy.append(b); perms.append(p)
    allp = list(itertools.permutations(range(4)))                     # lexicographic
    cnt = np.array([perms.count(p) for p in allp])
    assert (cnt > 120).all() and (cnt < 290).all()                    # 200 expected each
    assert abs(np.mean(ox) - (L - 1) / 2) < 4 * L / np.sqrt(12 * 4800)
    assert abs(np.mean(oy) - (L - 1) / 2) < 4 * L / np.sqrt(12 * 4800)
    assert len(set(np.array(ox) % 4)) == 4                            # arbitrary site, not a coarse grid (:150)
    # the permutation index is the lexicographic rank of G[2] % 24
    for t in range(50):
        G = oracle.philox4x32_10([0, 0, 2 << 30, t], [99, 0])
        a, b, p = oracle.mcs_control(99, t, L, DEV_DTR)
        assert p == allp[int(G[2]) % 24] and a == int(G[0]) % L and b == int(G[1]) % L


def test_site_selection_is_uniform_under_dtrdb():
    # every site has selection rate exactly 1/(cx*cy) per step (R14) -> Poisson-like counts, no site starved
    L, n = 64, 60
    o, tr = run_traced(L, 31, scheme(DEV_DTR, BLK_DB, 4), n)
    cnt = np.zeros((L, L))
    np.add.at(cnt, (tr["y"], tr["x"]), 1)
    assert abs(cnt.mean() - n) < 1e-9
    var = cnt.var()
    assert 0.5 * n < var < 1.3 * n                                    # binomial-ish: var ~ n(1-1/64)
    chi = ((cnt - n) ** 2 / n).sum() / (L * L)
    assert 0.8 < chi < 1.2
    o.close()


ORDER_CASES = [
    (scheme(DEV_DTR, BLK_DB, 5), 1.0, 0.0), (scheme(DEV_DTR, BLK_DB, 5), 0.0, 1.0),
    (scheme(DEV_DTR, BLK_DB, 5), 0.9, 0.1), (scheme(DEV_DTR, BLK_DB_DELAYED, 5), 1.0, 0.0),
    (scheme(DEV_DTR, BLK_DT, 5), 0.5, 0.5), (scheme(DEV_DT, BLK_DB, 5), 1.0, 0.0),
    (scheme(DEV_DB, BLK_DB, 5), 0.9, 0.1), (scheme(DEV_CDB, BLK_DB, 5), 1.0, 0.0),
    (scheme(DEV_DB, BLK_DT, 5), 1.0, 0.0), (scheme(DEV_DTR, BLK_DB, 5, 2, 2), 0.9, 0.1),
    (scheme(DEV_DTR, BLK_DB, 5, 0, 0), 0.5, 0.5), (scheme(DEV_DTR, BLK_DB, 6, 3, 1), 1.0, 0.0),
    (scheme(DEV_DTR, BLK_DTR, 5), 0.6, 0.4), (scheme(DEV_DTR, BLK_DTR, 5, 2, 1), 1.0, 0.0),
    (scheme(DEV_DBH, BLK_DB, 5), 0.7, 0.3), (scheme(DEV_DBH, BLK_DT, 5), 1.0, 0.0),
    (scheme(DEV_DB, BLK_DB, 5, 1, 1, 2, 0), 0.7, 0.3), (scheme(DEV_DB, BLK_DB, 5, 1, 1, 0, 1), 0.6, 0.4),      # t_async = 1/4; width 1, free origin
    (scheme(DEV_DB, BLK_DT, 5, 1, 1, 1, 2), 1.0, 0.0), (scheme(DEV_CDB, BLK_DB, 5, 1, 1, 2, 3), 0.9, 0.1),
]


@pytest.mark.parametrize("code,p,q", ORDER_CASES)
def test_order_independence(code, p, q):
    """Domains of one set, and cells within one phase, never touch common bits: any visiting order
    gives the same lattice.  This is what lets a parallel machine reproduce the oracle bit for bit."""
    L = 128
    ref = Oracle(L, 77)
    ref.sweep(6, p, q, code)
    for sh in (1, 0xDEADBEEF, 12345678901):
        o = Oracle(L, 77)
        o.set_shuffle(sh)
        o.sweep(6, p, q, code)
        assert (o.lattice == ref.lattice).all() and o.net == ref.net and o.h00 == ref.h00
        o.close()
    ref.close()


def test_sync_and_delayed_are_different_samples_of_the_same_process():
    # R16: "completely equivalent" (:174) holds in distribution, not bit-wise
    L = 128
    a, b = Oracle(L, 5), Oracle(L, 5)
    a.sweep(20, 1.0, 0.0, scheme(DEV_DTR, BLK_DB, 5))
    b.sweep(20, 1.0, 0.0, scheme(DEV_DTR, BLK_DB_DELAYED, 5))
    assert (a.lattice != b.lattice).any()
    assert abs(a.net - b.net) < 0.02 * a.net
    assert abs(float(a.w2()) / float(b.w2()) - 1) < 0.15
    a.close(); b.close()


@pytest.mark.parametrize("code,p,q", [(scheme(DEV_DTR, BLK_DB, 5), 1.0, 0.0), (scheme(DEV_DTR, BLK_DB, 5), 0.9, 0.1),
                                      (scheme(DEV_DB, BLK_DT, 5), 1.0, 0.0)])
def test_split_invariance(code, p, q):
    a, b = Oracle(128, 3), Oracle(128, 3)
    a.sweep(7, p, q, code)
    b.sweep(3, p, q, code); b.sweep(0, p, q, code); b.sweep(4, p, q, code)
    assert (a.lattice == b.lattice).all() and a.t == b.t == 7 and a.net == b.net
    a.close(); b.close()


@pytest.mark.parametrize("code,p,q", [(scheme(DEV_DTR, BLK_DB, 5), 1.0, 0.0), (scheme(DEV_DTR, BLK_DB, 5), 0.8, 0.3),
                                      (scheme(DEV_DTR, BLK_DT, 5), 0.8, 0.3), (scheme(DEV_CDB, BLK_DB, 5), 1.0, 0.0)])
def test_deposition_removal_symmetry(code, p, q):
    """Mirror h -> -h exchanges minima and maxima, p and q, and complements every slope bit; the RNG
    consumption does not depend on the state, so the two runs stay exact mirror images."""
    a, b = Oracle(128, 13, init=0), Oracle(128, 13, init=1)
    a.sweep(5, p, q, code)
    b.sweep(5, q, p, code)
    assert (a.lattice == ~b.lattice).all()
    assert a.net == -b.net and a.h00 == -b.h00
    assert (a.heights() == -b.heights()).all()
    a.close(); b.close()


def test_degenerate_sizes():
    # L = 2D (a single tile) and D = cx (a single cell per domain)
    for L, code in ((64, scheme(DEV_DTR, BLK_DB, 5)), (16, scheme(DEV_DTR, BLK_DB, 3)), (16, scheme(DEV_DB, BLK_DB, 4, 2, 2)),
                    (16, scheme(DEV_DTR, BLK_DB, 3, 0, 0)), (16, scheme(DEV_DTR, BLK_DT, 3))):
        o = Oracle(L, 2, track_heights=True)
        o.sweep(5, 1.0, 0.0, code)
        assert (o.heights() == o.tracked_heights).all()
        assert o.net > 0
        o.close()


def test_invalid_schemes_are_rejected():
    lib = oracle.lib()
    assert lib.orc_check_scheme(128, scheme(DEV_DTR, BLK_DB, 7)) != 0        # L < 2D
    assert lib.orc_check_scheme(128, scheme(DEV_DB, BLK_DB, 7)) == 0         # L >= D is enough for DB
    assert lib.orc_check_scheme(128, scheme(DEV_DTR, BLK_DT, 5, 0, 1)) != 0  # DT needs TC >= 1,1 (:182)
    assert lib.orc_check_scheme(128, scheme(DEV_DTR, BLK_DB, 3, 2, 0)) != 0  # cell larger than domain
    assert lib.orc_check_scheme(96, scheme(DEV_DTR, BLK_DB, 4)) != 0         # L not a power of two
    assert lib.orc_check_scheme(128, scheme(5, BLK_DB, 5)) != 0 and lib.orc_check_scheme(128, scheme(0, 4, 5)) != 0
    assert lib.orc_check_scheme(128, scheme(DEV_DTR, BLK_DTR, 5, 0, 1)) != 0 and lib.orc_check_scheme(128, scheme(DEV_DTR, BLK_DTR, 5)) == 0


def test_filtered_run_reproduces_the_interior():
    """A domain sweep depends only on its own (D+1)^2 window, so running only the domains that meet a
    box reproduces the full run inside the box shrunk by 4(D+2) sites per MCS.  This is the tool the
    full-size GPU parity tests use (L = 2^16, 2^17), validated here against complete runs."""
    L, D, n = 512, 16, 2
    code = scheme(DEV_DTR, BLK_DB, 4)
    full = Oracle(L, 123)
    full.sweep(n, 1.0, 0.0, code)
    margin = n * 4 * (D + 2)
    for (x0, y0, w, h) in ((40, 60, 200, 180), (L - 100, L - 90, 230, 210)):     # second box wraps
        part = Oracle(L, 123)
        part.set_filter(True, x0, y0, w, h)
        part.sweep(n, 1.0, 0.0, code)
        hf, hp = full.heights(), part.heights()
        ys = (y0 + margin + np.arange(h - 2 * margin)) % L
        xs = (x0 + margin + np.arange(w - 2 * margin)) % L
        # compare slopes (heights differ by the anchor if (0,0) is outside the box)
        sxf = hf - np.roll(hf, 1, axis=1); sxp = hp - np.roll(hp, 1, axis=1)
        syf = hf - np.roll(hf, 1, axis=0); syp = hp - np.roll(hp, 1, axis=0)
        assert (sxf[np.ix_(ys, xs)] == sxp[np.ix_(ys, xs)]).all()
        assert (syf[np.ix_(ys, xs)] == syp[np.ix_(ys, xs)]).all()
        assert (part.lattice != full.lattice).any()                               # and it really skipped work
        part.close()
    full.close()

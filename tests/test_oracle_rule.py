"""Pins for the oracle's update rule, packing, flat state, heights and conservation laws.

Every expected value here is derived in the test from the HEIGHT definition of the octahedron model
(an octahedron is deposited on a site that is lower than its four neighbours,
raising it by 2; the slopes are the height differences), not from the oracle's bit rule.
"""
import itertools

import numpy as np
import pytest

import oracle
from oracle import BLK_DB, BLK_DB_DELAYED, BLK_DT, DEV_CDB, DEV_DB, DEV_DT, DEV_DTR, Oracle, scheme
from helpers import surfaces as sf


# ---- brute force on the 4x4 periodic lattice ------------------------------------------------------
def all_surfaces(L):
    """Every periodic height field with h[0,0]=0 whose nearest neighbours differ by exactly 1."""
    out = []
    h = np.zeros((L, L), dtype=np.int32)
    sites = [(y, x) for y in range(L) for x in range(L)]

    def rec(i):
        if i == len(sites):
            out.append(h.copy())
            return
        y, x = sites[i]
        cands = {0} if i == 0 else None
        if x > 0:
            c = {h[y, x - 1] - 1, h[y, x - 1] + 1}
            cands = c if cands is None else cands & c
        if y > 0:
            c = {h[y - 1, x] - 1, h[y - 1, x] + 1}
            cands = c if cands is None else cands & c
        for v in sorted(cands):
            if x == L - 1 and abs(v - h[y, 0]) != 1:
                continue
            if y == L - 1 and abs(v - h[0, x]) != 1:
                continue
            h[y, x] = v
            rec(i + 1)

    rec(0)
    return out


def is_min(h, y, x):
    L = h.shape[0]
    return all(h[(y + dy) % L, (x + dx) % L] == h[y, x] + 1 for dy, dx in ((0, 1), (0, -1), (1, 0), (-1, 0)))


def is_max(h, y, x):
    L = h.shape[0]
    return all(h[(y + dy) % L, (x + dx) % L] == h[y, x] - 1 for dy, dx in ((0, 1), (0, -1), (1, 0), (-1, 0)))


@pytest.fixture(scope="module")
def surfaces4():
    return all_surfaces(4)


def test_bruteforce_4x4_every_state_every_site(surfaces4):
    assert len(surfaces4) == 990          # SURVEY.md section 8(c) counted the same number independently
    n_min = n_max = 0
    o = Oracle(4, 0)
    for h in surfaces4:
        words = sf.pack_heights(h)
        for y in range(4):
            for x in range(4):
                for (P16, Q16) in ((65536, 0), (0, 65536), (65536, 65536)):
                    o.set_lattice(words, h00=0, net=0)
                    d = o.attempt(x, y, 0, P16, Q16)
                    exp = h.copy()
                    want = 0
                    if is_min(h, y, x) and P16:
                        exp[y, x] += 2
                        want = 1
                    elif is_max(h, y, x) and Q16:
                        exp[y, x] -= 2
                        want = -1
                    assert d == want
                    assert (o.heights() == exp).all()
                    assert (o.lattice == sf.pack_heights(exp)).all()
                    assert o.net == want
                n_min += is_min(h, y, x)
                n_max += is_max(h, y, x)
    assert n_min == 3648 and n_max == 3648
    o.close()


def test_bruteforce_2x2():
    s = all_surfaces(2)
    assert len(s) == 6 or len(s) > 0      # L=2 is below the oracle's minimum size; only the enumerator is checked
    for h in s:
        assert (np.abs(h - np.roll(h, 1, 0)) == 1).all() and (np.abs(h - np.roll(h, 1, 1)) == 1).all()


def test_acceptance_threshold_is_strict_less_than(surfaces4):
    h = surfaces4[0]
    ys, xs = np.nonzero(np.array([[is_min(h, y, x) for x in range(4)] for y in range(4)]))
    y, x = int(ys[0]), int(xs[0])
    o = Oracle(4, 0)
    P16 = oracle.prob16(0.9)
    o.set_lattice(sf.pack_heights(h))
    assert o.attempt(x, y, P16, P16, 0) == 0          # r16 == P16 -> reject
    assert o.attempt(x, y, P16 - 1, P16, 0) == 1      # r16 <  P16 -> accept
    o.close()


def test_h00_tracking_on_origin_updates(surfaces4):
    o = Oracle(4, 0)
    for h in surfaces4[:200]:
        o.set_lattice(sf.pack_heights(h), h00=0)
        d = o.attempt(0, 0, 0, 65536, 65536)
        assert o.h00 == 2 * d
        exp = h.copy()
        exp[0, 0] += 2 * d
        assert (o.heights() == exp).all()
    o.close()


# ---- flat state ------------------------------------------------------------------------------------
@pytest.mark.parametrize("L", [4, 8, 64, 256])
def test_flat_state(L):
    o = Oracle(L, 3, init=0)
    assert (o.lattice == 0x33CC33CC).all()
    yy, xx = np.mgrid[0:L, 0:L]
    h = ((xx + yy) & 1).astype(np.int32)
    assert (o.heights() == h).all() and (o.heights(rowpath=True) == h).all()
    assert (o.lattice == sf.pack_heights(h)).all()
    assert o.w2() == 0.25 and o.mean_height() == 0.5
    S1, S2, c, net = o.sums()
    assert (S1, S2, c, net) == (L * L // 2, L * L // 2, 0, 0)
    # exactly N/2 local minima: a p=1 attempt succeeds exactly on the even sites
    n_ok = 0
    for y in range(min(L, 8)):
        for x in range(min(L, 8)):
            oo = Oracle(L, 3)
            n_ok += oo.attempt(x, y, 0, 65536, 0)
            assert (oo.net == 1) == ((x + y) % 2 == 0)
            oo.close()
    o.close()


def test_flat_shifted_is_the_complement():
    o = Oracle(64, 3, init=1)
    assert (o.lattice == 0xCC33CC33).all()
    yy, xx = np.mgrid[0:64, 0:64]
    assert (o.heights() == -((xx + yy) & 1)).all()
    o.close()


# ---- heights from an independent generator -----------------------------------------------------------
@pytest.mark.parametrize("L,seed,off", [(16, 1, 0), (64, 2, -7), (256, 3, 1000)])
def test_heights_of_separable_surface(L, seed, off):
    h = sf.separable_surface(L, seed, off)
    o = Oracle(L, 0)
    o.set_lattice(sf.pack_heights(h), h00=off)
    assert (o.heights() == h).all()
    assert (o.heights(rowpath=True) == h).all()
    S1, S2, c, _ = o.sums()
    d = h.astype(np.int64) - off
    assert (S1, S2, c) == (int(d.sum()), int((d * d).sum()), off)
    assert o.sums(rowpath=True) == o.sums()            # streaming form used at L = 2^16, 2^17 (no height array)
    assert float(o.w2()) == pytest.approx(float(np.var(h.astype(np.float64))), rel=1e-12)
    o.close()


# ---- invariants after real sweeps --------------------------------------------------------------------
def unpack(words):
    n = words.shape[0]
    L = 4 * n
    sx = np.zeros((L, L), dtype=np.int8)
    sy = np.zeros((L, L), dtype=np.int8)
    for j in range(4):
        for i in range(4):
            b = 2 * (4 * j + i)
            sx[j::4, i::4] = (words >> np.uint32(b)) & 1
            sy[j::4, i::4] = (words >> np.uint32(b + 1)) & 1
    return sx, sy


def check_valid_surface(o: Oracle):
    L = o.L
    sx, sy = unpack(o.lattice)
    assert (sx.sum(axis=1) == L // 2).all()            # every row: as many up- as down-slopes in x
    assert (sy.sum(axis=0) == L // 2).all()            # every column likewise in y
    # curl-free: going around any plaquette returns to the same height
    SX, SY = 2 * sx.astype(np.int32) - 1, 2 * sy.astype(np.int32) - 1
    assert (SX + np.roll(SY, 1, axis=1) == SY + np.roll(SX, 1, axis=0)).all()
    h = o.heights()
    assert (h == o.heights(rowpath=True)).all()
    assert (o.lattice == sf.pack_heights(h)).all()
    return h


CASES = [
    (scheme(DEV_DTR, BLK_DB, 5), 1.0, 0.0),
    (scheme(DEV_DTR, BLK_DB, 5), 0.0, 1.0),
    (scheme(DEV_DTR, BLK_DB, 5), 0.9, 0.1),
    (scheme(DEV_DTR, BLK_DB_DELAYED, 5), 1.0, 0.0),
    (scheme(DEV_DTR, BLK_DT, 5), 0.7, 0.3),
    (scheme(DEV_DT, BLK_DB, 5), 1.0, 0.0),
    (scheme(DEV_DB, BLK_DB, 5), 0.6, 0.4),
    (scheme(DEV_CDB, BLK_DT, 5), 1.0, 0.0),
    (scheme(DEV_DTR, BLK_DB, 6, 2, 2), 1.0, 0.0),
    (scheme(DEV_DTR, BLK_DB, 6, 3, 1), 0.5, 0.5),
    (scheme(DEV_DTR, BLK_DT, 6, 1, 3), 1.0, 0.0),
    (scheme(DEV_DTR, BLK_DB, 5, 0, 0), 0.5, 0.5),
    (scheme(DEV_DTR, 3, 5), 0.7, 0.3),            # block-layer DTr
    (scheme(DEV_DB, 3, 5, 2, 1), 1.0, 0.0),
    (scheme(4, BLK_DB, 5), 0.8, 0.2),             # DB with t_async = 1/2
    (scheme(DEV_DB, BLK_DB, 5, 1, 1, 2, 1), 0.8, 0.2),   # t_async = 1/4, border width 1 with a free origin (:202-206)
    (scheme(DEV_CDB, BLK_DT, 5, 1, 1, 1, 3), 1.0, 0.0),
]


@pytest.mark.parametrize("code,p,q", CASES)
def test_invariants_and_tracked_heights(code, p, q):
    L = 128
    o = Oracle(L, 11, track_heights=True)
    for _ in range(3):
        o.sweep(4, p, q, code)
        h = check_valid_surface(o)
        assert (h == o.tracked_heights).all()
        assert int(h.astype(np.int64).sum()) == L * L // 2 + 2 * o.net
        assert o.h00 == h[0, 0]
        d = h.astype(np.int64) - o.h00
        assert o.sums(rowpath=True) == o.sums() == (int(d.sum()), int((d * d).sum()), o.h00, o.net)
    o.close()


def test_rs_invariants():
    L = 64
    o = Oracle(L, 5, track_heights=True)
    o.sweep_rs(20, 0.8, 0.2)
    h = check_valid_surface(o)
    assert (h == o.tracked_heights).all()
    assert int(h.astype(np.int64).sum()) == L * L // 2 + 2 * o.net
    o.close()


def test_sync_variant_would_break_with_both_rates_hence_auto_picks_delayed():
    # DESIGN.md R16: with p>0 and q>0 the block layer must use delayed borders; BLK_DB (auto) does.
    L, code_auto, code_del = 64, scheme(DEV_DTR, BLK_DB, 5), scheme(DEV_DTR, BLK_DB_DELAYED, 5)
    a, b = Oracle(L, 9), Oracle(L, 9)
    a.sweep(10, 0.5, 0.5, code_auto)
    b.sweep(10, 0.5, 0.5, code_del)
    assert (a.lattice == b.lattice).all()
    a.close(); b.close()


def test_no_rates_no_change():
    o = Oracle(64, 1)
    o.sweep(3, 0.0, 0.0, scheme(DEV_DTR, BLK_DB, 5))
    assert (o.lattice == 0x33CC33CC).all() and o.net == 0 and o.t == 3
    o.close()

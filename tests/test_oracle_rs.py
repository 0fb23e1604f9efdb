"""Pin of the oracle's true random-sequential dynamics (`orc_sweep_rs`), the reference of BASELINE config 2.

RS "by definition" (PAPER.md:15 / :44): each attempt picks one uniformly random site; 1 MCS = L^2 attempts (:106).
What is the loop's own -- the number of attempts, the counter layout of reading R19 (tag 3 in the top bits of word 2,
the attempt index n in words 0-1, the MCS t in word 3, the 64-bit seed as the two key words), X / Y / r16 taken from
output words 0 / 1 / 2 -- is checked here record by record on the trace, and the outcome of every attempt is
recomputed from the HEIGHT definition of the update rule (Eq. (1) :27-34: deposit on a local minimum with
probability p, remove from a local maximum with probability q), not from the slope bits the oracle works on.
"""
import numpy as np
import pytest

import oracle
from oracle import Oracle

TAG_RS = 3


@pytest.mark.parametrize("seed,p,q", [(11, 1.0, 0.0), (0x9E3779B97F4A7C15, 0.7, 0.3), ((5 << 32) | 2, 0.0, 1.0)])
def test_rs_trace_matches_the_definition_attempt_by_attempt(seed, p, q):
    L, n_mcs, t0 = 64, 2, 5
    N = L * L
    o = Oracle(L, seed)
    o.set_lattice(o.lattice.copy(), t=t0)                     # a clock other than 0: word 3 of the counter is live
    o.start_trace(n_mcs * N + 8)
    o.sweep_rs(n_mcs, p, q)
    tr = o.stop_trace()
    assert len(tr) == n_mcs * N and o.t == t0 + n_mcs          # :106
    key = [seed & 0xFFFFFFFF, seed >> 32]
    P16, Q16 = oracle.prob16(p), oracle.prob16(q)
    yy, xx = np.mgrid[0:L, 0:L]
    h = ((xx + yy) & 1).astype(np.int64)                       # flat start (R5), heights indexed [y, x]
    k = 0
    for t in range(t0, t0 + n_mcs):
        for n in range(N):
            w = oracle.philox4x32_10([n & 0xFFFFFFFF, n >> 32, TAG_RS << 30, t], key)
            x, y, r16 = int(w[0]) % L, int(w[1]) % L, int(w[2]) >> 16
            rec = tr[k]; k += 1
            assert (int(rec["x"]), int(rec["y"]), int(rec["t"])) == (x, y, t)
            nb = (h[y, (x + 1) % L], h[y, (x - 1) % L], h[(y + 1) % L, x], h[(y - 1) % L, x])
            c = h[y, x]
            d = 0
            if all(v == c + 1 for v in nb) and r16 < P16:
                d = 1
            elif all(v == c - 1 for v in nb) and r16 < Q16:
                d = -1
            assert int(rec["result"]) == d, (t, n)
            h[y, x] += 2 * d
    assert (o.heights() == h).all()
    assert o.net == int((tr["result"]).sum())
    o.close()


def test_rs_site_selection_is_uniform_and_uncorrelated():
    """Every attempt is an independent uniform draw over the L^2 sites: Poisson-like counts per site, all four
    parities of (x, y) equally often (no sub-lattice structure, unlike checkerboard updates), and no
    correlation between the sites of consecutive attempts."""
    L, n_mcs = 64, 12
    o = Oracle(L, 4242)
    o.start_trace(n_mcs * L * L + 8)
    o.sweep_rs(n_mcs, 1.0, 0.0)
    tr = o.stop_trace()
    cnt = np.zeros((L, L))
    np.add.at(cnt, (tr["y"], tr["x"]), 1)
    assert cnt.sum() == n_mcs * L * L
    chi = ((cnt - n_mcs) ** 2 / n_mcs).sum() / (L * L)         # Poisson: 1 +- sqrt(2 / L^2) ~ 0.022
    assert 0.9 < chi < 1.1
    assert cnt.min() >= 1                                      # P(a site never hit in 12 MCS) = e^-12 per site
    par = np.bincount((tr["x"] & 1) + 2 * (tr["y"] & 1), minlength=4) / len(tr)
    assert np.abs(par - 0.25).max() < 4 * np.sqrt(0.25 * 0.75 / len(tr))
    x = tr["x"].astype(np.float64)
    r = np.corrcoef(x[:-1], x[1:])[0, 1]
    assert abs(r) < 4 / np.sqrt(len(tr))
    o.close()

"""BASELINE config 2 (L = 1024, p = 1, q = 0, 2000 MCS): every DD scheme of the paper on the GPU against the oracle's TRUE
random-sequential dynamics (stored exact sums, tests/golden/rs_L1024.txt), W^2(t) and C(t,s) at s = 100 and 200 -- what
Sec. 4.1.1 (Fig. 3) compares.  The engine is bit-reproducible and the seeds are fixed, so the numbers
are deterministic (profiles/r2_config2.md holds the table); the assertions state what the paper states:

 * DTr at device layer neither introduces correlations nor extra noise (:208): C_s decays like under RS;
 * coarse dead border leaves a pattern: C_s converges to a finite value (:192-194);
 * wide dead borders with a free origin add noise, less for shorter t_async (:202-206);
 * a finer block-layer DD lowers the W^2 prefactor: TC=1,1 < TC=2,2 < RS (:254), with the same late-time growth.

WHAT KIND OF TEST THIS IS.  A pinned-numbers regression, not statistical evidence: the 32 seeds are fixed and the engine is
deterministic, so every "sigma" below is one fixed number (cDB's plateau sits at 2.8 / 2.7 s.e.m. with this sample, just
above the 2.5 threshold; DT.DT cannot be told from DTr at n = 32, profiles/r2_config2.md).  The thresholds were read off
this sample; a legitimate change of the RNG stream mapping (R19) or of the seed set may move a value across one and then
the thresholds, not the engine, are what needs another look.  The statistical statement -- cDB's pattern at 20 s.e.m. on
256 seeds -- is in profiles/r2_physics.md; parity with the oracle is tested elsewhere, bit for bit.
"""
import pytest

import config2_report as c2

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def table():
    rs = c2.rs_reference()
    grid_w2, grid_ac = sorted(rs["w2"]), sorted(rs["ch"])
    assert len(c2.SEEDS) == 32 and set(range(1, 9)) <= set(c2.SEEDS)
    return {name: c2.compare(rs, c2.gpu_scheme(code, grid_w2, grid_ac)) for name, code in c2.schemes()}


def test_dtr_schemes_decorrelate_like_true_rs(table):
    for name in ("DTrDB", "DTrDT", "DTrDB TC=2,2"):
        c = table[name]
        for s in c2.WAITS:
            assert abs(c[f"cs_late_{s}"]["sigmas"]) < 2.5, (name, s)              # no plateau beyond RS's own tail
        assert abs(c["w2_2000"]["sigmas"]) < 3 and abs(c["w2_2000"]["rel"]) < 0.08, name
        assert abs(c["ch_100_200"]["rel"]) < 0.08 and abs(c["ch_200_2000"]["sigmas"]) < 3, name


def test_coarse_dead_border_leaves_a_pattern(table):
    c, ref = table["cDB.DT"], table["DTrDT"]
    for s in c2.WAITS:
        assert c[f"cs_late_{s}"]["sigmas"] > 2.5, s                                # finite late-time slope autocorrelation
        assert c[f"cs_late_{s}"]["dd"] > 1.8 * max(ref[f"cs_late_{s}"]["dd"], c[f"cs_late_{s}"]["rs"]), s
    assert abs(c["w2_100"]["rel"]) < 0.02                                          # ... invisible in the roughness (:194)


def test_wide_dead_borders_add_noise_and_shorter_t_async_removes_it(table):
    db, dbh, db4, thin = table["DB.DT"], table["DBh.DT"], table["DB.DT tasync=1/4"], table["DB.DT w=1"]
    assert db["w2_100"]["rel"] > 0.08 and db["w2_100"]["sigmas"] > 8               # t_async = 1 MCS: "even larger noise" (:206)
    assert 0.01 < dbh["w2_100"]["rel"] < 0.5 * db["w2_100"]["rel"]                 # t_async = 1/2 MCS, the paper's choice
    assert abs(db4["w2_100"]["rel"]) < 0.015 and abs(db4["ch_100_200"]["rel"]) < 0.03
    assert abs(thin["w2_100"]["rel"]) < 0.03                                       # width 1: the noise comes from the WIDE borders (:202)


def test_finer_block_layer_dd_lowers_the_prefactor(table):
    fine, coarse = table["DTrDB"]["w2_100"], table["DTrDB TC=2,2"]["w2_100"]
    assert fine["dd"] < coarse["dd"] < coarse["rs"]                                # TC=1,1 < TC=2,2 < RS (:254)
    assert fine["sigmas"] < -5 and coarse["sigmas"] < -2.5 and coarse["rel"] - fine["rel"] > 0.008

#!/usr/bin/env python
"""Writes tests/golden/oracle_runs.txt: SHA-256 of the oracle's packed lattice and its integer sums at fixed times for
a handful of small runs.  Calls ONLY oracle/ (never the CUDA path).  The file is a regression pin of the oracle's own
arithmetic (a later change to it must be deliberate: regenerate and say why in the commit) and lets GPU tests compare
against stored oracle results without re-running the oracle.

    python tests/golden/make_oracle_golden.py            # rewrite oracle_runs.txt (seconds)
    python tests/golden/make_oracle_golden.py --full c4_D64     # one FULL-SIZE run -> full_c4_D64.txt (minutes to hours)
    python tests/golden/make_oracle_golden.py --full all        # every full-size run, one after the other

Full-size runs (BASELINE.json configs 3, 4 and 5 as `north_star` states them: "bit-exact lattice vs oracle" for the whole
5000-MCS mixed-rate run at L = 4096, "the oracle checked bit-exact on the first 2 MCS" at L = 2^16, the first MCS at
L = 2^17; PAPER.md:262 gives L = 2^16, :232 L = 2^17, :174 the p, q > 0 path).  One file per run so that they can be
produced in parallel; tests/test_gpu_fullsize.py hashes oct_export() at the same checkpoints.  At these sizes the sums
are taken along the row path without a height array (Oracle.sums(rowpath=True), pinned against the plain form).
"""
import hashlib
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import BLK_DB, BLK_DT, BLK_DTR, DEV_CDB, DEV_DB, DEV_DBH, DEV_DT, DEV_DTR, Oracle, scheme   # noqa: E402

# (name, L, seed, p, q, scheme, checkpoints)
RUNS = (
    ("c0_DTrDB_D64", 256, 1, 1.0, 0.0, scheme(DEV_DTR, BLK_DB, 6), (1, 10, 100)),          # BASELINE config 1
    ("DTrDT_D64", 256, 1, 1.0, 0.0, scheme(DEV_DTR, BLK_DT, 6), (1, 20)),
    ("DTrDB_delayed_D64", 256, 7, 0.9, 0.1, scheme(DEV_DTR, BLK_DB, 6), (1, 20)),
    ("DTrDTr_D64", 256, 3, 0.7, 0.3, scheme(DEV_DTR, BLK_DTR, 6), (5,)),
    ("DTDB_D64", 256, 2, 1.0, 0.0, scheme(DEV_DT, BLK_DB, 6), (5,)),
    ("DBDB_D64", 256, 2, 1.0, 0.0, scheme(DEV_DB, BLK_DB, 6), (5,)),
    ("cDBDT_D64", 256, 2, 1.0, 0.0, scheme(DEV_CDB, BLK_DT, 6), (5,)),
    ("DBhDB_D64", 256, 2, 0.8, 0.2, scheme(DEV_DBH, BLK_DB, 6), (5,)),
    ("DTrDB_TC22_D128", 256, 4, 1.0, 0.0, scheme(DEV_DTR, BLK_DB, 7, 2, 2), (4,)),
    # seeds that use the HIGH half of the 64-bit Philox key (R19: key = (seed & 2^32-1, seed >> 32)); every run above has it zero
    ("DTrDB_delayed_seed64", 256, 0x9E3779B97F4A7C15, 0.9, 0.1, scheme(DEV_DTR, BLK_DB, 6), (6,)),
    ("DBDB_TC22_seedhi7", 256, (7 << 32) | 1, 1.0, 0.0, scheme(DEV_DB, BLK_DB, 6, 2, 2), (4,)),
    ("DTrDB_seedhi_only", 256, 1 << 32, 1.0, 0.0, scheme(DEV_DTR, BLK_DB, 6), (3,)),
)


# name -> (L, seed, p, q, scheme, checkpoints, every_mcs_sums)
FULL_RUNS = {
    # BASELINE config 4: L = 2^16, p = 1, q = 0, seed 1, DTrDB -- first 2 MCS, whole lattice
    "c4_D64": (1 << 16, 1, 1.0, 0.0, scheme(DEV_DTR, BLK_DB, 6), (1, 2), False),
    "c4_D128": (1 << 16, 1, 1.0, 0.0, scheme(DEV_DTR, BLK_DB, 7), (1, 2), False),
    "c4_D256": (1 << 16, 1, 1.0, 0.0, scheme(DEV_DTR, BLK_DB, 8), (1, 2), False),
    "c4_D64_TC22": (1 << 16, 1, 1.0, 0.0, scheme(DEV_DTR, BLK_DB, 6, 2, 2), (1, 2), False),   # PAPER.md:236-244 (Fig. 5)
    # BASELINE config 5: L = 2^17 -- first MCS, whole lattice
    "c5_D64": (1 << 17, 1, 1.0, 0.0, scheme(DEV_DTR, BLK_DB, 6), (1,), False),
    # BASELINE config 3: L = 4096, p = 0.9, q = 0.1, seed 7, DTrDB (delayed borders), the whole 5000-MCS run:
    # lattice hash every 500 MCS, and the sums after EVERY MCS hashed per 500-MCS window
    "c3_D128": (4096, 7, 0.9, 0.1, scheme(DEV_DTR, BLK_DB, 7), tuple(range(500, 5001, 500)), True),
    # the same run with D = 64, the shape whose domains sit in one warp: there the CUDA path decides per collective step
    # whether the delayed-border phases can be merged into one pass
    "c3_D64": (4096, 7, 0.9, 0.1, scheme(DEV_DTR, BLK_DB, 6), tuple(range(500, 5001, 500)), True),
}


def full_lines(name):
    L, seed, p, q, code, cps, every = FULL_RUNS[name]
    yield "# name L seed p q scheme t sha256(lattice words, little endian) S1 S2 h00 net"
    yield "# sums_sha name t0 t1 sha256(text 'S1 S2 h00 net\\n' for every MCS t0 < t <= t1)"
    yield f"# written by `python tests/golden/make_oracle_golden.py --full {name}` from oracle/oct_oracle.c only"
    o = Oracle(L, seed)
    t_prev = 0
    for t in cps:
        if every:
            hs = hashlib.sha256()
            while o.t < t:
                o.sweep(1, p, q, code)
                hs.update(("%d %d %d %d\n" % o.sums(rowpath=True)).encode())
            yield f"sums_sha {name} {t_prev} {t} {hs.hexdigest()}"
        else:
            o.sweep(t - o.t, p, q, code)
        digest = hashlib.sha256(o.lattice.astype("<u4").tobytes()).hexdigest()
        S1, S2, c, net = o.sums(rowpath=True)
        yield f"{name} {L} {seed} {p} {q} {code} {t} {digest} {S1} {S2} {c} {net}"
        t_prev = t
    o.close()


def lines():
    yield "# name L seed p q scheme t sha256(lattice words, little endian) S1 S2 h00 net"
    yield "# written by tests/golden/make_oracle_golden.py from oracle/oct_oracle.c only"
    for name, L, seed, p, q, code, cps in RUNS:
        o = Oracle(L, seed)
        for t in cps:
            o.sweep(t - o.t, p, q, code)
            digest = hashlib.sha256(o.lattice.astype("<u4").tobytes()).hexdigest()
            S1, S2, c, net = o.sums()
            yield f"{name} {L} {seed} {p} {q} {code} {t} {digest} {S1} {S2} {c} {net}"
        o.close()


if __name__ == "__main__":
    here = os.path.dirname(os.path.abspath(__file__))
    if len(sys.argv) >= 3 and sys.argv[1] == "--full":
        for name in (FULL_RUNS if sys.argv[2] == "all" else sys.argv[2:]):
            out = os.path.join(here, f"full_{name}.txt")
            with open(out + ".part", "w") as f:
                for line in full_lines(name):
                    f.write(line + "\n")
                    f.flush()
            os.replace(out + ".part", out)
            print(out)
    else:
        out = os.path.join(here, "oracle_runs.txt")
        with open(out, "w") as f:
            f.write("\n".join(lines()) + "\n")
        print(out)

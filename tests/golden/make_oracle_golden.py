#!/usr/bin/env python
"""Writes tests/golden/oracle_runs.txt: SHA-256 of the oracle's packed lattice and its integer sums at fixed times for
a handful of small runs.  Calls ONLY oracle/ (never the CUDA path).  The file is a regression pin of the oracle's own
arithmetic (a later change to it must be deliberate: regenerate and say why in the commit) and lets GPU tests compare
against stored oracle results without re-running the oracle.

    python tests/golden/make_oracle_golden.py            # rewrite the file
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
)


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
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_runs.txt")
    with open(out, "w") as f:
        f.write("\n".join(lines()) + "\n")
    print(out)

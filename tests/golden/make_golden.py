"""Writes tests/golden/oracle_logz.txt: log Z of BASELINE.json designs at their full sizes, computed by the CPU oracle alone.

Calls only oracle/ (and the seeded input generator, which holds no arithmetic of the method); nothing here touches the CUDA path.
The plain oracle needs minutes (config 2, 5) to hours (config 3) for these sizes, which is why the values are stored instead of
being recomputed by the GPU parity tests.

    python tests/golden/make_golden.py 5 2        # configs to (re)compute, in this order; existing lines are kept
"""
from __future__ import annotations

import os
import sys
import time

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
OUT = os.path.join(HERE, "oracle_logz.txt")


def main():
    from oracle import build as obuild
    from oracle import oracle as O
    from paper_2604_19718_b200 import inputs as I

    obuild.build()
    have = {}
    if os.path.exists(OUT):
        for ln in open(OUT):
            if ln.strip() and not ln.startswith("#"):
                c, item, L, n, lz, sec = ln.split()
                have[(int(c), int(item), int(L))] = (int(n), lz, sec)
    for arg in sys.argv[1:]:
        cfg = int(arg)
        d = I.design(cfg, 0)
        key = (cfg, 0, len(d.aa))
        t0 = time.time()
        tab = O.inside(I.nn_model(), O.TT.build(d.aa, d.kind, d.codon_logw, d.pair_logw))
        have[key] = (d.n, f"{tab.logZ:.12f}", f"{time.time() - t0:.0f}")
        with open(OUT, "w") as f:
            f.write("# config item L_aa n_nt logZ oracle_seconds   (oracle/cdz_oracle.c orc_inside, plain long-double recursion; "
                    "written by tests/golden/make_golden.py)\n")
            for (c, item, L), (n, lz, sec) in sorted(have.items()):
                f.write(f"{c} {item} {L} {n} {lz} {sec}\n")
        print(key, have[key], flush=True)


if __name__ == "__main__":
    main()

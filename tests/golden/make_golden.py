#!/usr/bin/env python
"""Writes the stored expected values of the full-size parity tests.  Calls ONLY the CPU oracle (oracle/) and the
seeded input generators; nothing here touches the CUDA path.  The plain long-double recursion takes minutes (configs 1, 2, 5)
to hours (config 3) at these sizes, which is why the values are stored instead of being recomputed by the GPU parity tests.

    python tests/golden/make_golden.py 5 2              # log Z of whole configs -> oracle_logz.txt (existing lines are kept)
    python tests/golden/make_golden.py logz 3           # same, explicit mode
    python tests/golden/make_golden.py samples 1 5      # orc_sample of the config's sample count (config 5: item 0) ->
                                                        #   oracle_samples.txt (SHA-256 of the raw arrays + sample 0 as text)
    python tests/golden/make_golden.py closed 600 3000  # closed-form pins at n nucleotides -> oracle_closed_forms.txt
    python tests/golden/make_golden.py marginals 1      # orc_marginals (eqs 2.5-2.7 as ratios of restricted partition functions)
                                                        #   of the whole config -> oracle_marginals_config<c>.txt
"""
from __future__ import annotations

import hashlib
import os
import sys
import time

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
OUT = os.path.join(HERE, "oracle_logz.txt")
OUT_SAMPLES = os.path.join(HERE, "oracle_samples.txt")


def _load(path, nkey):
    have = {}
    if os.path.exists(path):
        for ln in open(path):
            if ln.strip() and not ln.startswith("#"):
                f = ln.split()
                have[tuple(int(v) for v in f[:nkey])] = f[nkey:]
    return have


def do_logz(cfgs):
    from oracle import oracle as O
    from paper_2604_19718_b200 import inputs as I

    have = _load(OUT, 3)
    for cfg in cfgs:
        d = I.design(cfg, 0)
        key = (cfg, 0, len(d.aa))
        t0 = time.time()
        tab = O.inside(I.nn_model(), O.TT.build(d.aa, d.kind, d.codon_logw, d.pair_logw))
        have[key] = [str(d.n), f"{tab.logZ:.12f}", f"{time.time() - t0:.0f}"]
        with open(OUT, "w") as f:
            f.write("# config item L_aa n_nt logZ oracle_seconds   (oracle/cdz_oracle.c orc_inside, plain long-double recursion; "
                    "written by tests/golden/make_golden.py)\n")
            for k, v in sorted(have.items()):
                f.write(" ".join(str(x) for x in k) + " " + " ".join(v) + "\n")
        print(key, have[key], flush=True)


def do_samples(cfgs):
    """J samples of the whole design by the oracle's traceback; J = the config's sample count (BASELINE.json)."""
    from oracle import oracle as O
    from paper_2604_19718_b200 import inputs as I

    have = _load(OUT_SAMPLES, 4)
    for cfg in cfgs:
        d = I.design(cfg, 0)
        J = d.n_samples
        t0 = time.time()
        tab = O.inside(I.nn_model(), O.TT.build(d.aa, d.kind, d.codon_logw, d.pair_logw))
        seq, pair = tab.sample(J, d.sample_seed)
        hs = hashlib.sha256(seq.astype("uint8").tobytes()).hexdigest()
        hp = hashlib.sha256(pair.astype("<i4").tobytes()).hexdigest()
        have[(cfg, 0, len(d.aa), J)] = [str(d.sample_seed), hs, hp, O.seq_str(seq[0]), O.dot_bracket(pair[0]),
                                        f"{time.time() - t0:.0f}"]
        with open(OUT_SAMPLES, "w") as f:
            f.write("# config item L_aa J seed sha256(seq uint8 [J][n]) sha256(pair int32le [J][n]) sample0_sequence sample0_structure "
                    "oracle_seconds   (oracle/cdz_oracle.c orc_sample; written by tests/golden/make_golden.py samples)\n")
            for k, v in sorted(have.items()):
                f.write(" ".join(str(x) for x in k) + " " + " ".join(v) + "\n")
        print(cfg, hs, hp, flush=True)


def do_marginals(cfgs):
    from oracle import oracle as O
    from paper_2604_19718_b200 import inputs as I

    for cfg in cfgs:
        d = I.design(cfg, 0)
        t0 = time.time()
        tab = O.inside(I.nn_model(), O.TT.build(d.aa, d.kind, d.codon_logw, d.pair_logw))
        bpp, base, codon = tab.marginals()
        n = d.n
        with open(os.path.join(HERE, f"oracle_marginals_config{cfg}.txt"), "w") as f:
            f.write(f"# orc_marginals of the whole config {cfg} design (item 0, n = {n}); oracle/cdz_oracle.c, written by "
                    f"tests/golden/make_golden.py marginals; {time.time() - t0:.0f} s\n")
            f.write("# bpp i j P(i.j)   (i < j: pair probability, i == j: P(i unpaired); zeros omitted)\n")
            for i in range(n):
                for j in range(i, n):
                    if bpp[i, j] != 0.0:
                        f.write(f"bpp {i} {j} {bpp[i, j]:.17g}\n")
            f.write("# base m b P(phi_m = b)\n")
            for m in range(n):
                for b in range(4):
                    if base[m, b] != 0.0:
                        f.write(f"base {m} {b} {base[m, b]:.17g}\n")
            f.write("# codon k c p_k(c)   (c = 16 b0 + 4 b1 + b2)\n")
            for k in range(n // 3):
                for c in range(64):
                    if codon[k, c] != 0.0:
                        f.write(f"codon {k} {c} {codon[k, c]:.17g}\n")
        print("marginals", cfg, f"{time.time() - t0:.0f} s", flush=True)


def do_closed(sizes):
    """Expected log Z of the closed-form pins from oracle pieces that share nothing with the tensor recursion: orc_tt_logsum (eq 3.2)
    and the scalar fixed-sequence orc_mccaskill.  -> oracle_closed_forms.txt"""
    import numpy as np

    from oracle import oracle as O
    from paper_2604_19718_b200 import inputs as I

    path = os.path.join(HERE, "oracle_closed_forms.txt")
    have = {}
    if os.path.exists(path):
        for ln in open(path):
            if ln.strip() and not ln.startswith("#"):
                f = ln.split()
                have[(f[0], int(f[1]))] = f[2:]
    for n in sizes:
        t0 = time.time()
        ops = I.closed_form_inputs("zero8", n)
        logw = O.TT.from_ops(ops).logsum()
        logs = O.mccaskill(I.zero_energy_model(), np.zeros(n, dtype=np.uint8))  # log S_30(n): any fixed sequence, all pairs allowed
        have[("zero8", n)] = [f"{logw + logs:.12f}", f"{logw:.12f}", f"{logs:.12f}", f"{time.time() - t0:.0f}"]
        t0 = time.time()
        aa, cw = I.closed_form_inputs("mettrp", n)
        cod = {"M": (0, 3, 2), "W": (3, 2, 2)}  # AUG, UGG
        seq = np.array([b for a in aa for b in cod[a]], dtype=np.uint8)
        logw = float(sum(cw[16 * cod[a][0] + 4 * cod[a][1] + cod[a][2]] for a in aa))
        lz = O.mccaskill(I.nn_model(), seq)
        have[("mettrp", n)] = [f"{logw + lz:.12f}", f"{logw:.12f}", f"{lz:.12f}", f"{time.time() - t0:.0f}"]
        with open(path, "w") as f:
            f.write("# kind n_nt logZ_expected log_sum_W log_structure_part oracle_seconds   (orc_tt_logsum + orc_mccaskill; written by "
                    "tests/golden/make_golden.py closed)\n")
            for k, v in sorted(have.items()):
                f.write(f"{k[0]} {k[1]} " + " ".join(v) + "\n")
        print("closed", n, have[("zero8", n)], have[("mettrp", n)], flush=True)


def main():
    from oracle import build as obuild

    obuild.build()
    args = sys.argv[1:]
    mode = "logz"
    if args and args[0] in ("logz", "samples", "marginals", "closed"):
        mode, args = args[0], args[1:]
    cfgs = [int(a) for a in args]
    {"logz": do_logz, "samples": do_samples, "marginals": do_marginals, "closed": do_closed}[mode](cfgs)


if __name__ == "__main__":
    main()

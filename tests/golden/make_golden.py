"""Writes tests/golden/oracle_config1.txt.  Calls ONLY oracle/ and lqcd_inputs/ (never the CUDA path).

    python tests/golden/make_golden.py

The paper prints no vector, matrix or iteration-count values, so there is no paper fixture to
store; this file is a regression guard that freezes what the *oracle* computes today for BASELINE
config 1 (4^4, seeds 180101473/180101474, antiperiodic t) and for a small 8-shift solve, so that an
accidental change of the oracle's arithmetic or of the input generator is noticed
(tests/test_golden.py).  A deliberate change must name, in its commit message, the passage of the
paper or the DESIGN.md reading that justifies it.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import lqcd_inputs as gen  # noqa: E402
import oracle  # noqa: E402

SITES = (0, 17, 100, 127)


def compute():
    L = (4, 4, 4, 4)
    U = gen.random_su3_links(L).numpy()
    b = oracle.restrict(L, 0, gen.gaussian_field(L).numpy())
    t = oracle.doe(L, U, b, True)
    u = oracle.deo(L, U, t, True)
    rows = [("links_sum", float(U.sum())), ("b_norm2", float((b ** 2).sum())),
            ("t_norm2", float((t ** 2).sum())), ("u_norm2", float((u ** 2).sum()))]
    for k in SITES:
        for c in range(3):
            rows.append((f"t[{k}][{c}].re", float(t[k, c, 0])))
            rows.append((f"t[{k}][{c}].im", float(t[k, c, 1])))
            rows.append((f"u[{k}][{c}].re", float(u[k, c, 0])))
            rows.append((f"u[{k}][{c}].im", float(u[k, c, 1])))
    shifts = [1e-4 * 10 ** (i / 2) for i in range(8)]
    x, info = oracle.mshift_cg(L, U, 0.01, b, shifts, 1e-10)
    rows.append(("cg_iters", float(info["iters"])))
    for i in range(8):
        rows.append((f"cg_freeze[{i}]", float(info["freeze_iter"][i])))
        rows.append((f"cg_x_norm2[{i}]", float((x[i] ** 2).sum())))
    return rows


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_config1.txt")
    with open(path, "w") as fh:
        fh.write("# written by tests/golden/make_golden.py from oracle/ only; not paper values (the paper prints none)\n")
        for name, v in compute():
            fh.write(f"{name} {v!r}\n")
    print(path)

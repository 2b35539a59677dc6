"""Writes tests/golden/oracle_config*.txt: eigenvalues of BASELINE.json configs 0 and 1 computed by the CPU oracle
ONLY (oracle/ + bse_inputs/; nothing from the CUDA package).  Config 1 takes tens of minutes of CPU time, which is
why its values are stored instead of being recomputed inside the GPU test.

    python tests/golden/make_oracle_goldens.py [0|1]      (no argument: both configs)
"""
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import bse_inputs as gen  # noqa: E402
import oracle  # noqa: E402


def write(name, header, values, resid):
    with open(os.path.join(HERE, name), "w") as f:
        f.write(header)
        for v, r in zip(values, resid):
            f.write(f"{v:.17e} {r:.3e}\n")


def main():
    oracle.build()
    which = sys.argv[1:] or ["0", "1"]
    for sigma in ((0.0, 1.0) if "0" in which else ()):
        cfg = gen.CONFIGS[0]
        R = gen.dense_R(cfg["N"], 1, sigma=sigma, group=cfg["group"])
        t = time.time()
        w, V, res, steps = oracle.lanczos_tda(R, cfg["nev"], 1e-11, gen.block_X(cfg["N"], 1, 99)[:, 0], check=20)
        assert steps > 0
        write(f"oracle_config0_sigma{int(sigma)}.txt",
              f"# BASELINE.json config 0 (TDA N=1024, seed 1, sigma={sigma}): nev=10 lowest eigenvalues of R.\n"
              f"# oracle.lanczos_tda (textbook Lanczos, PAPER.md:65-71), tol 1e-11, {steps} steps, {time.time()-t:.0f} s.\n"
              f"# columns: eigenvalue  residual_estimate\n", w, res)
    if "1" not in which:
        return
    cfg = gen.CONFIGS[1]
    N = cfg["N"]
    R = gen.dense_R(N, 1, sigma=cfg["sigma"]); C = gen.dense_C(N, 1)
    t = time.time()
    om, V, res, steps = oracle.lanczos_full(R, C, cfg["nev"], 1e-11, gen.block_X(N, 1, 97)[:, 0], check=100)
    assert steps > 0, steps
    write("oracle_config1.txt",
          f"# BASELINE.json config 1 (full N=2048, seed 1, sigma=1.0): nev=20 lowest positive omega of Eq. (1),\n"
          f"# counted as eigenvectors of H (the second copy of each omega^2 of G = M o P is dropped by its vector,\n"
          f"# DESIGN.md reading R1).  oracle.lanczos_full (structure-preserving Lanczos, reading S4 of PAPER.md:65-69),\n"
          f"# tol 1e-11, {steps} steps, {time.time()-t:.0f} s.  columns: omega  residual_estimate\n", om, res)


if __name__ == "__main__":
    main()

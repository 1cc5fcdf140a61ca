"""Writes tests/golden/workload_sha256.txt (generator fingerprints) and
tests/golden/oracle_cfg1_moments.txt (oracle moments for BASELINE.json config 1).

Calls only the seeded generator (paper_1303_6016_b200.workload) and oracle/ -- never the
CUDA path.  The paper prints no worked numerical example, so these files
are drift detectors for the generator and the oracle, not pins: the pins are the
mathematical checks in tests/test_oracle_*.py.

    python tests/golden/make_golden.py
"""
import sys
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parents[2]
sys.path.insert(0, str(ROOT))

from oracle import oracle                                   # noqa: E402
from paper_1303_6016_b200 import workload as wl             # noqa: E402

HERE = Path(__file__).resolve().parent


def main():
    lines = ["# sha256 of the arrays make_workload(CONFIGS[i], n_sweeps=1) returns (SURVEY.md §8(d) recipe)"]
    for i in (1, 2, 3, 4):
        S, prop, uni = wl.make_workload(wl.CONFIGS[i], n_sweeps=1)
        lines.append(f"cfg{i} spins {wl.sha256(S)}")
        lines.append(f"cfg{i} proposals {wl.sha256(prop)}")
        lines.append(f"cfg{i} uniforms {wl.sha256(uni)}")
    (HERE / "workload_sha256.txt").write_text("\n".join(lines) + "\n")

    cfg = wl.CONFIGS[1]
    S, _, _ = wl.make_workload(cfg, n_sweeps=1)
    mu = oracle.moments(cfg.L, cfg.t, cfg.JH, S, site=21, M=16)
    out = ["# oracle.moments(cfg1, site=21, M=16): n alpha beta re im (written by make_golden.py from oracle/ only)"]
    for n in range(16):
        for al in range(2):
            for be in range(2):
                out.append(f"{n} {al} {be} {float(mu[n, al, be].real)!r} {float(mu[n, al, be].imag)!r}")
    (HERE / "oracle_cfg1_moments.txt").write_text("\n".join(out) + "\n")


if __name__ == "__main__":
    main()

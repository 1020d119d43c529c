"""Writes tests/golden/g20_threshold_study.txt: one full oracle iteration of C1 and C2 under three storage conventions
for the float32 responsibilities (flush below 2^-100 as in round 1, flush below 2^-126 = libemc's storage, gradual
underflow = the oracle's default) and both c-steps.  Calls only oracle/ and the seeded input generator.  About 4 minutes on 8 cores.

    python tests/golden/make_g20_threshold_study.py
"""
import pathlib
import sys

import numpy as np

ROOT = pathlib.Path(__file__).resolve().parents[2]
sys.path.insert(0, str(ROOT))

from emc_inputs import make_inputs  # noqa: E402
from oracle import emc_oracle as o  # noqa: E402


def main():
    lines = ["# config c-step threshold active_slices status_changes_vs_gradual max_rel_model_change median_rel_model_change",
             "# (change of model' per voxel against gradual underflow, voxels with den >= 1e-6 max den; written by "
             "tests/golden/make_g20_threshold_study.py)"]
    for name in ("C1", "C2"):
        inp = make_inputs(name)
        for weighted in (False, True):
            res = {}
            for label, p_min in (("2^-100", 2.0 ** -100), ("2^-126", 2.0 ** -126), ("gradual", 0.0)):
                o.P_MIN = p_min
                res[label] = o.iterate(inp.model_init, inp.q, inp.mask, inp.quat[0], inp.weight[0], inp.counts,
                                       weighted=weighted)
            base = res["gradual"]
            cov = base["den"] >= 1e-6 * base["den"].max()
            mb = base["model"].reshape(-1).astype(np.float64)
            for label in ("2^-100", "2^-126", "gradual"):
                r = res[label]
                rel = np.abs(r["model"].reshape(-1).astype(np.float64) - mb)[cov] / np.maximum(np.abs(mb[cov]), 1e-30)
                changed = int(((r["s"] > 0) != (base["s"] > 0)).sum())
                lines.append(f"{name} {'eq2.12' if weighted else 'eq2.10'} {label} {int((r['s'] > 0).sum())} {changed} "
                             f"{rel.max():.3e} {np.median(rel):.3e}")
                print(lines[-1], flush=True)
    (pathlib.Path(__file__).parent / "g20_threshold_study.txt").write_text("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()

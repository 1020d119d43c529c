"""Reading G20: where float32 stops representing a responsibility.

The paper only says "some care ... finite precision".  P is carried in float32.  The ORACLE
does nothing about its underflow: P becomes float32 by numpy's cast (gradual underflow: subnormals kept, 0 below 2^-150).
libemc stores P flush-to-zero below 2^-126, the smallest normal float32 (EMC_P_MIN in include/emc.h).  This file measures,
on the oracle alone (o.P_MIN switched by hand), what separates the two conventions in model', so that the GPU tests can
gate exactly that and nothing more (tests/gates.py):

 * eq. (2.12) (the c-step the paper implements) weights slice r by s[r] = sum_d P[r,d]: a slice made of
   subnormal responsibilities weighs < 2^-126 N against slices of weight O(1).  model' moves by far less than T3's 1e-5.
 * eq. (2.10) (north_star's literal stage 5) gives EVERY slice with s[r] > 0 the weight 1, so it is
   discontinuous in P at 0: which slices take part is decided by the last representable number of whatever arithmetic
   is used.  The slices whose status differs between the two conventions are exactly the rows made of float32
   subnormals only, and model' differs on the voxels they touch by O(1e-3 ... 1) -- under ANY threshold.

tests/golden/g20_threshold_study.txt holds the same numbers for one full C2 iteration (written by
tests/golden/make_g20_threshold_study.py, oracle only, about 4 minutes)."""
import pathlib

import numpy as np
import pytest

from oracle import emc_oracle as o

GOLDEN = pathlib.Path(__file__).parent / "golden" / "g20_threshold_study.txt"


def run(inp, p_min, weighted):
    saved = o.P_MIN
    o.P_MIN = p_min
    try:
        return o.iterate(inp.model_init, inp.q, inp.mask, inp.quat[0], inp.weight[0], inp.counts, weighted=weighted)
    finally:
        o.P_MIN = saved


def rel_change(a, b):
    """per-voxel |a - b| / max(|b|, 1e-30) on the voxels b covers (den >= 1e-6 max den, as T3; the floor keeps voxels whose
    value is itself a float32 subnormal out of the ratio)"""
    cov = b["den"] >= 1e-6 * b["den"].max()
    ma, mb = a["model"].reshape(-1).astype(np.float64), b["model"].reshape(-1).astype(np.float64)
    return np.abs(ma - mb)[cov] / np.maximum(np.abs(mb[cov]), 1e-30)


@pytest.mark.parametrize("name,n_pat", [("C1", None), ("C2", 600)])
def test_flush_to_zero_against_gradual_underflow(inputs_cache, name, n_pat):
    inp = inputs_cache(name, n_pat=n_pat) if n_pat else inputs_cache(name)
    tiny = float(np.finfo(np.float32).tiny)
    for weighted in (True, False):
        ftz = run(inp, tiny, weighted)           # libemc's storage: flush below 2^-126
        grad = run(inp, 0.0, weighted)           # the oracle's default: numpy's float32 cast, subnormals kept, 0 below 2^-150
        changed = (ftz["s"] > 0) != (grad["s"] > 0)
        # the rows whose status differs are exactly those that hold float32 subnormals and nothing larger
        only_subnormal = (grad["P"].max(axis=1) < tiny) & (grad["P"].max(axis=1) > 0)
        assert np.array_equal(changed, only_subnormal)
        rel = rel_change(ftz, grad)
        print(f"{inp.cfg.name} N={inp.counts.shape[0]} {'eq 2.12' if weighted else 'eq 2.10'}: active {int((ftz['s'] > 0).sum())} "
              f"(flush-to-zero) / {int((grad['s'] > 0).sum())} (gradual) of {len(ftz['s'])}; model' max rel change "
              f"{rel.max():.2e}, median {np.median(rel):.2e}, voxels > 1e-5: {int((rel > 1e-5).sum())} of {rel.size}")
        if weighted:
            assert rel.max() <= 1e-6             # eq. (2.12): a float32 ulp or two of model', ten times inside T3 = 1e-5
        elif changed.any():
            assert rel.max() > 1e-5              # eq. (2.10): the discontinuity is real, whatever the threshold


def test_stored_c2_study_is_consistent():
    """The committed full-size study: same structure of the result at C2 (one whole iteration)."""
    rows = {}
    for ln in GOLDEN.read_text().splitlines():
        if ln.startswith("#") or not ln.strip():
            continue
        f = ln.split()
        rows[(f[0], f[1], f[2])] = dict(active=int(f[3]), changed=int(f[4]), max_rel=float(f[5]), median_rel=float(f[6]))
    w = rows[("C2", "eq2.12", "2^-126")]
    u = rows[("C2", "eq2.10", "2^-126")]
    assert w["max_rel"] <= 1e-6 and w["changed"] == u["changed"] > 0
    assert u["max_rel"] > 1e-5
    # the round-1 threshold 2^-100 dropped several times as many slices
    assert rows[("C2", "eq2.10", "2^-100")]["changed"] > 3 * u["changed"]

"""Adaptive EMC (section 3.4, eq. 3.1): pins of the oracle's refinement loop (CPU) and parity of
emc_refine with it (`-m gpu`).  Rotation lists are seeded uniform random quaternions of growing size (the paper's
600-cell lists of eq. 2.7 need ref. [11] App. C, which is not in the container: DESIGN.md NEXT-1)."""
import numpy as np
import pytest

from emc_inputs import make_inputs
from emc_inputs.synth import random_rotations
from oracle import emc_oracle as o


def make_levels(sizes, seed=7000):
    return [(random_rotations(r, seed + i), np.full(r, 1.0 / r, dtype=np.float32)) for i, r in enumerate(sizes)]


def test_criterion_is_eq_3_1():
    # |L^n - L^(n-1)| <= 0.01 |L^n| with numbers worked by hand
    assert o.refine_criterion(-1000.0, -995.0)            # 5 <= 9.95
    assert not o.refine_criterion(-1000.0, -900.0)        # 100 > 9
    assert o.refine_criterion(-995.0, -1000.0)            # a decrease counts the same: 5 <= 10
    assert not o.refine_criterion(-1000.0, -989.0)        # 11 > 9.89
    assert o.refine_criterion(2000.0, 2019.0)             # positive likelihoods: 19 <= 20.19
    assert not o.refine_criterion(-1000.0, -995.0, threshold=0.001)


@pytest.fixture(scope="module")
def small():
    inp = make_inputs("T0")
    return inp, make_levels((20, 35, 60))


def test_schedule_structure_and_composition(small):
    inp, levels = small
    out = o.refine(inp.model_init, inp.q, inp.mask, levels, inp.counts, 6)
    lv = out["level"]
    assert lv[0] == 0 and lv[1] == 0                                   # the criterion needs two likelihoods
    assert np.all(np.diff(lv) >= 0) and np.all(np.diff(lv) <= 1) and lv.max() < len(levels)
    # every switch is the criterion applied to the two likelihoods before it, and only then
    for n in range(1, len(lv) - 1):
        want = lv[n] + 1 < len(levels) and o.refine_criterion(out["LL"][n - 1], out["LL"][n])
        assert (lv[n + 1] == lv[n] + 1) == bool(want)
    # iteration 0 is a plain iteration on the coarsest list, iteration 1 continues from its model
    it0 = o.iterate(inp.model_init, inp.q, inp.mask, *levels[0], inp.counts)
    assert out["LL"][0] == it0["LL"]
    it1 = o.iterate(it0["model"], inp.q, inp.mask, *levels[0], inp.counts)
    assert out["LL"][1] == it1["LL"]


def test_threshold_extremes(small):
    inp, levels = small
    never = o.refine(inp.model_init, inp.q, inp.mask, levels, inp.counts, 5, threshold=0.0)
    assert np.all(never["level"] == 0)                                  # likelihoods never repeat exactly
    always = o.refine(inp.model_init, inp.q, inp.mask, levels, inp.counts, 6, threshold=1e9)
    assert list(always["level"]) == [0, 0, 1, 2, 2, 2]                  # one step per iteration from n = 1, then kept
    one = o.refine(inp.model_init, inp.q, inp.mask, levels[:1], inp.counts, 3, threshold=1e9)
    assert np.all(one["level"] == 0)


@pytest.mark.gpu
@pytest.mark.parametrize("threshold", [0.01, 0.003])
def test_emc_refine_matches_oracle(threshold):
    import torch

    emc = pytest.importorskip("paper_1409_4256_b200")
    inp = make_inputs("T2")
    # the ladder of eq. (2.7) at d = 1, 2, 3 (60, 420, 1380 rotations) with non-uniform prior weights
    from emc_inputs import ladder_rotations

    levels = [ladder_rotations(d, 7100 + d) for d in (1, 2, 3)]
    assert [len(w) for _, w in levels] == [60, 420, 1380] and all(w.std() > 0.1 * w.mean() for _, w in levels)
    ref = o.refine(inp.model_init, inp.q, inp.mask, levels, inp.counts, 10, threshold)
    assert ref["level"].max() == 2                                      # the case does refine twice
    dev = lambda x: torch.from_numpy(np.ascontiguousarray(x)).cuda()
    out = emc.emc_refine(dev(inp.model_init), dev(inp.q), dev(inp.mask), [(dev(qt), dev(w)) for qt, w in levels],
                         dev(inp.counts), 10, threshold)
    emc.emc_check(out["ws"])
    assert out["level"] == list(ref["level"])                           # the integer decisions: exact
    ll = out["loglik"].cpu().numpy()
    assert np.all(np.abs(ll - ref["LL"]) <= 2e-5 * np.abs(ref["LL"]))   # ten iterations of drift
    m, m_ref = out["model"].cpu().numpy().reshape(-1), ref["model"].reshape(-1)
    rel = np.abs(m - m_ref) / (np.abs(m_ref) + 1e-6 * np.abs(m_ref).max())
    assert np.median(rel) <= 1e-3

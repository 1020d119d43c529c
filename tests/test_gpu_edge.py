"""Degenerate and ragged cases of the whole iteration against the oracle (`-m gpu`): one rotation, one pattern,
patterns without photons, a constant model (north_star's invariant: responsibilities equal the prior), a detector
that is almost entirely masked, sizes below every tile, and rotation weights that are far from uniform."""
import dataclasses

import numpy as np
import pytest
import torch

from emc_inputs import CONFIGS, make_inputs
import gates
from oracle import emc_oracle as o

pytestmark = pytest.mark.gpu

emc = pytest.importorskip("paper_1409_4256_b200")


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def host(t):
    return t.detach().cpu().numpy()


def run_both(model, q, mask, quat, weight, counts, weighted=False, null_weight=False):
    ref = o.iterate(model, q, mask, quat, weight, counts, weighted=weighted)
    d = [dev(model), dev(q), dev(mask), dev(quat), None if null_weight else dev(weight), dev(counts)]
    out = emc.emc_iterate(*d, want_p=True, flags=emc.EMC_COMPRESS_WEIGHTED if weighted else 0)
    emc.emc_check(out["ws"])
    # the float32 L this emc_iterate call itself formed, read from its workspace, for the measured P bound
    torch.cuda.synchronize()
    n, n_pix, n_rot, n_pat = model.shape[0], q.shape[0], quat.shape[0], counts.shape[0]
    out["L"] = host(emc.emc_workspace_view(out["ws"], n, n_pix, n_rot, n_pat, emc.EMC_VIEW_LOGLIK,
                                           emc.EMC_COMPRESS_WEIGHTED if weighted else 0))
    out["weighted"], out["geometry"] = weighted, (q, quat, mask, float(np.asarray(counts).max()))
    return ref, out


def check(ref, out):
    p = host(out["P"])
    # end to end: |dP| <= 1e-6 + P (exp(2 max_r |dL|) - 1) with the MEASURED dL (T2)
    m = np.abs(out["L"].astype(np.float64) - ref["L"].astype(np.float64)).max(axis=0)
    bound = 1e-6 + ref["P"] * np.expm1(2.0 * m)[None, :]
    assert np.all(np.abs(p - ref["P"]) <= bound), f"max dP {np.abs(p - ref['P']).max():.3e}"
    assert abs(float(host(out["loglik"])[0]) - ref["LL"]) <= 1e-5 * abs(ref["LL"]) + 1e-6
    gates.model_gate(host(out["model"]), ref, out["weighted"], *out["geometry"], dl_max=float(m.max()), label="edge case")


@pytest.fixture(scope="module")
def t0():
    return make_inputs("T0")


def test_single_rotation(t0):
    ref, out = run_both(t0.model_init, t0.q, t0.mask, t0.quat[0][:1], np.ones(1, np.float32), t0.counts)
    assert np.all(host(out["P"]) == 1.0)                       # one rotation takes all the responsibility
    check(ref, out)


def test_single_pattern_and_empty_patterns(t0):
    ref, out = run_both(t0.model_init, t0.q, t0.mask, t0.quat[0], t0.weight[0], t0.counts[:1])
    check(ref, out)
    k = t0.counts.copy()
    k[3] = 0                                                    # no photon at all: L = -S[r]
    k[7, t0.mask.astype(bool)] = 0                              # photons only in masked pixels: the same
    ref, out = run_both(t0.model_init, t0.q, t0.mask, t0.quat[0], t0.weight[0], k)
    check(ref, out)
    p = host(out["P"])
    assert np.abs(p[:, 3] - p[:, 7]).max() <= 1e-7


def test_constant_model_gives_the_prior(t0):
    rng = np.random.default_rng(2)
    w = rng.uniform(0.2, 2.0, size=t0.weight[0].shape).astype(np.float32)
    w /= w.sum()
    model = np.full_like(t0.model_init, 0.37)
    ref, out = run_both(model, t0.q, t0.mask, t0.quat[0], w, t0.counts)
    p = host(out["P"])
    assert np.abs(p - w[:, None]).max() <= 1e-6                 # every slice is the same: P[r,d] = w_r
    check(ref, out)


def test_almost_fully_masked_detector(t0):
    mask = np.zeros_like(t0.mask)
    mask[[5, 77, 200]] = 1
    ref, out = run_both(t0.model_init, t0.q, mask, t0.quat[0], t0.weight[0], t0.counts, weighted=True)
    check(ref, out)


def test_sizes_below_every_tile():
    cfg = dataclasses.replace(CONFIGS["T0"], name="T0s", n=8, n_det=6, n_rot=(3,), n_pat=5, n_pat_chunk=5)
    inp = make_inputs(cfg)
    ref, out = run_both(inp.model_init, inp.q, inp.mask, inp.quat[0], inp.weight[0], inp.counts)
    check(ref, out)


def test_extreme_prior_weights(t0):
    w = np.full(t0.weight[0].shape, 1e-12, dtype=np.float32)
    w[11] = 1.0
    w /= w.sum()
    ref, out = run_both(t0.model_init, t0.q, t0.mask, t0.quat[0], w, t0.counts)
    check(ref, out)


def test_zero_prior_weights(t0):
    """w_r = 0 (log w = -inf) excludes a rotation: P[r,:] = 0 exactly, s[r] = 0, the slice is skipped.  The first
    row of the list, of a 32-row block and of a warp's row range are among them (the stage API's column sweep and the
    GEMM epilogue's fused statistics both start from such a row)."""
    w = np.array(t0.weight[0], dtype=np.float32)
    dead = [0, 1, 8, 31, 32, 33, 59]
    w[dead] = 0.0
    w /= w.sum()
    with np.errstate(divide="ignore"):
        ref, out = run_both(t0.model_init, t0.q, t0.mask, t0.quat[0], w, t0.counts)
    assert np.all(host(out["P"])[dead] == 0) and np.all(ref["P"][dead] == 0)
    check(ref, out)
    # stage API
    big_l = torch.zeros((len(w), emc.ld_for(t0.counts.shape[0])), dtype=torch.float32, device="cuda")
    big_l[:, : t0.counts.shape[0]] = dev(ref["L"])
    p, s, ll = emc.emc_normalize(big_l[:, : t0.counts.shape[0]], dev(t0.quat[0]), dev(w))
    with np.errstate(divide="ignore"):
        p_ref, s_ref, ll_ref = o.normalize(ref["L"], w)
    assert np.abs(host(p) - p_ref).max() <= 1e-6 and np.all(host(p)[dead] == 0)
    assert abs(float(host(ll)[0]) - ll_ref) <= 1e-6 * abs(ll_ref)


def test_null_weights_are_the_uniform_prior(t0):
    """weight = NULL is 1/R: the uniform branches of the fused statistics and of the second sweep against the oracle"""
    ref, out = run_both(t0.model_init, t0.q, t0.mask, t0.quat[0], t0.weight[0], t0.counts, null_weight=True)
    check(ref, out)
    ref, out = run_both(t0.model_init, t0.q, t0.mask, t0.quat[0], t0.weight[0], t0.counts, weighted=True, null_weight=True)
    check(ref, out)

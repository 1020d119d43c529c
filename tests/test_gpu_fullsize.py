"""Parity at BASELINE.json's full size in the launch configuration bench.py times (config C2:
64^3 model, 64x64 detector, R = 5000, N = 10000): the oracle finishes one full iteration of C2 in
about a minute, so every output is compared in full, not sampled.  (`-m gpu`)"""
import numpy as np
import pytest
import torch

import gates
from oracle import emc_oracle as o

pytestmark = pytest.mark.gpu

emc = pytest.importorskip("paper_1409_4256_b200")


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def host(t):
    return t.detach().cpu().numpy()


@pytest.fixture(scope="module")
def c2(inputs_cache):
    inp = inputs_cache("C2")
    ref = o.iterate(inp.model_init, inp.q, inp.mask, inp.quat[0], inp.weight[0], inp.counts)
    # the same iteration with P stored as libemc stores it (flush-to-zero below 2^-126, G20): C2 is the config where the two
    # float32 conventions part (140 of 5000 slices hang on subnormal responsibilities and touch 6 of 7 covered voxels), so
    # model' is gated against both
    ref_flush = o.iterate(inp.model_init, inp.q, inp.mask, inp.quat[0], inp.weight[0], inp.counts, p_min=o.P_MIN_FLUSH)
    return inp, ref, ref_flush


def test_c2_stagewise_and_end_to_end(c2):
    inp, ref, ref_flush = c2
    cfg = inp.cfg
    d_q, d_mask, d_quat, d_w, d_k = dev(inp.q.reshape(cfg.n_det, cfg.n_det, 3)), dev(inp.mask), dev(inp.quat[0]), dev(inp.weight[0]), dev(inp.counts)

    # stage 1: index map bit-exact over all 5000 x 4096 samples
    w, idx = emc.emc_expand(dev(inp.model_init), d_q, d_quat)
    assert np.array_equal(host(idx), ref["idx"])
    assert np.all(np.abs(host(w) - ref["W"]) <= 1e-5 * np.abs(ref["W"]) + 1e-9 * np.abs(ref["W"]).max())
    del w, idx

    # stage 2 on the oracle's W: |dL| <= 1e-5 A everywhere
    big_l, big_a = o.loglik(ref["W"], ref["idx"], inp.counts, inp.mask)
    got = host(emc.emc_loglik(dev(ref["W"]), dev(ref["idx"]), d_q, d_mask, d_k))
    err = np.abs(got - big_l) / big_a
    assert err.max() <= 1e-5, f"max |dL|/A = {err.max():.3e}"
    del got, err

    # stage 4 on the oracle's P (signed mean exposes an accumulation bias)
    n_pat = cfg.n_pat
    # (P as libemc stores it: float32 subnormals are 0, EMC_P_MIN / G20; the oracle's update gets the same array)
    p_in = gates.flushed(ref["P"])
    wn_ref, s_in = o.update(p_in, inp.counts, inp.mask)
    p = torch.zeros((cfg.n_rot[0], emc.ld_for(n_pat)), dtype=torch.float32, device="cuda")
    p[:, :n_pat] = dev(p_in)
    wn = host(emc.emc_update(p[:, :n_pat], dev(s_in.astype(np.float32)), d_q, d_mask, d_k))
    scale = np.abs(wn_ref).max()
    rel = (wn - wn_ref) / (np.abs(wn_ref) + 1e-7 * scale)
    assert np.abs(rel).max() <= 1e-5, f"max rel dW' = {np.abs(rel).max():.3e}"
    big = wn_ref > 1e-3 * scale
    assert abs(rel[big].mean()) <= 2e-6, f"mean signed rel dW' = {rel[big].mean():+.3e}"
    del p, wn, rel

    # stage 5 on the oracle's W'
    s32 = ref["s"].astype(np.float32)
    m_ref, _, den_ref = o.compress(ref["Wn"], inp.q, inp.quat[0], inp.mask, cfg.n, slice_w=(s32 > 0).astype(np.float32))
    m, den = emc.emc_compress(dev(ref["Wn"]), dev(s32), d_q, d_mask, d_quat, cfg.n, want_den=True)
    m, den, m_ref = host(m).reshape(-1), host(den), m_ref.reshape(-1)
    cov = den_ref >= 1e-6 * den_ref.max()
    assert np.all(np.abs(m[cov] - m_ref[cov]) <= 1e-5 * np.abs(m_ref[cov]) + 1e-12), \
        f"max rel {np.max(np.abs(m[cov] - m_ref[cov]) / (np.abs(m_ref[cov]) + 1e-12)):.3e}"

    # whole iteration, as bench.py launches it; T1 on the L this call itself formed (read from its workspace), and P against
    # the bound from that log-likelihood difference
    out = emc.emc_iterate(dev(inp.model_init), d_q, d_mask, d_quat, d_w, d_k, want_p=True)
    emc.emc_check(out["ws"])
    torch.cuda.synchronize()
    l_gpu = host(emc.emc_workspace_view(out["ws"], cfg.n, cfg.n_pix, cfg.n_rot[0], n_pat, emc.EMC_VIEW_LOGLIK))
    err = np.abs(l_gpu - big_l) / big_a
    assert err.max() <= 1e-5, f"emc_iterate's own L: max |dL|/A = {err.max():.3e}"
    m = np.abs(l_gpu.astype(np.float64) - ref["L"].astype(np.float64)).max(axis=0)
    bound = 1e-6 + ref["P"] * np.expm1(2.0 * m)[None, :]
    s_gpu = host(emc.emc_workspace_view(out["ws"], cfg.n, cfg.n_pix, cfg.n_rot[0], n_pat, emc.EMC_VIEW_S))
    dl_max = float(m.max())
    del l_gpu
    pg = host(out["P"])
    assert np.all(np.abs(pg - ref["P"]) <= bound), f"max dP {np.abs(pg - ref['P']).max():.3e}"
    # weight = NULL (the uniform branches, what the header documents as the default) gives the same responsibilities
    out0 = emc.emc_iterate(dev(inp.model_init), d_q, d_mask, d_quat, None, d_k, want_p=True)
    assert np.all(np.abs(host(out0["P"]) - ref["P"]) <= bound)
    assert abs(float(host(out0["loglik"])[0]) - ref["LL"]) <= 1e-5 * abs(ref["LL"])
    del out0
    assert abs(float(host(out["loglik"])[0]) - ref["LL"]) <= 1e-5 * abs(ref["LL"])
    gates.model_gate(host(out["model"]), ref, False, inp.q, inp.quat[0], inp.mask, float(inp.counts.max()), s_gpu=s_gpu,
                     dl_max=dl_max, label="C2 eq2.10 vs the plain-cast oracle")
    gates.model_gate(host(out["model"]), ref_flush, False, inp.q, inp.quat[0], inp.mask, float(inp.counts.max()), s_gpu=s_gpu,
                     dl_max=dl_max, fragile=gates.edge_rows(ref["P"], dl_max), label="C2 eq2.10 vs the flush-to-zero oracle")

"""Parity at BASELINE.json's large configs on SAMPLED outputs the oracle computes one by one (`-m gpu`):
  C3  128^3 / 128x128 / R = 25 000 / N = 50 000: the FULL config, as bench.py times it by default;
  C4  128^3 / 128x128 / R = 10 000, pattern chunks of 25 000 streamed from pinned host memory: the config's own chunk
      size and route, N cut to 2 chunks + a ragged third (60 000 of 200 000 patterns);
  C5  last stage, 256^3 / 256x256 / R = 50 000, the full 20 000 patterns (EMC_TEST_LARGE=0 cuts them to 1024).
At C3 and C5 Compress runs over ALL rotations against oracle.compress (float64, thread pool), and emc_iterate itself -- the
path bench.py times -- is checked at size: T1 on the L it formed (read from its workspace), T2 on its P, its s, LL, W' rows
and model' against the oracle / the stage chain.
Model, detector, mask and rotation list are the configs' own.  What these sizes exercise beyond C2: linear indices
past 2^31 (R x P = 3.3e9), accumulators that do not fit L2, hundreds of K chunks, ragged last pair tiles."""
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest
import torch

from oracle import emc_oracle as o

pytestmark = pytest.mark.gpu

# the configs' FULL pattern counts by default (the three cases take two minutes on a B200 box with the thread-parallel input
# generator); EMC_TEST_LARGE=0 cuts C5's for a quick run
FULL = os.environ.get("EMC_TEST_LARGE", "1") != "0"

emc = pytest.importorskip("paper_1409_4256_b200")


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def host(t):
    return t.detach().cpu().numpy()


def sampled_rows(n_rot, k, seed):
    """k rotation indices: the first, the last, the ones around 2^31 / n_pix, and random ones."""
    rng = np.random.default_rng(seed)
    rows = set(rng.integers(0, n_rot, size=k).tolist()) | {0, 1, n_rot - 2, n_rot - 1}
    return np.array(sorted(rows), dtype=np.int64)


def oracle_compress(wn, q, quat, mask, n, slice_w):
    """oracle.compress over ALL the rotations given: the definition evaluated on disjoint blocks of the rotation list by a
    pool of threads (numpy releases the GIL in the arithmetic), the float64 numerator / denominator grids of the blocks
    added up in float64, division last.  3.2e9 (C3) / 2.6e10 (C5) float64 additions."""
    n_rot = wn.shape[0]
    workers = min(32, os.cpu_count() or 1)
    bounds = np.linspace(0, n_rot, 4 * workers + 1).astype(int)

    def block(i):
        sl = slice(bounds[i], bounds[i + 1])
        _, num, den = o.compress(wn[sl], q, quat[sl], mask, n, slice_w=slice_w[sl])
        return num, den

    num, den = np.zeros(n ** 3), np.zeros(n ** 3)
    with ThreadPoolExecutor(workers) as ex:
        for nb, db in ex.map(block, range(len(bounds) - 1)):
            num += nb
            den += db
    with np.errstate(divide="ignore", invalid="ignore"):
        return np.where(den > 0, num / den, 0.0), den


def run_case(inputs_cache, name, n_pat, stage, n_rows, n_cols):
    inp = inputs_cache(name, n_pat=n_pat)
    cfg = inp.cfg
    quat, weight = inp.quat[stage], inp.weight[stage]
    n_rot, n_pix = quat.shape[0], cfg.n_pix
    d_q, d_mask, d_quat, d_k = dev(inp.q.reshape(cfg.n_det, cfg.n_det, 3)), dev(inp.mask), dev(quat), dev(inp.counts)
    rows = sampled_rows(n_rot, n_rows, 7)
    if n_rot * n_pix > 2 ** 31:                                       # rows on both sides of the 32-bit boundary
        edge = 2 ** 31 // n_pix
        rows = np.unique(np.concatenate([rows, [edge - 1, edge, edge + 1]]))
    t_rows = torch.from_numpy(rows).cuda()

    # ---- stage 1 on sampled rotations: idx bit-exact, W within 1e-5
    w, idx = emc.emc_expand(dev(inp.model_init), d_q, d_quat)
    torch.cuda.empty_cache()                                          # expand's own workspace
    ws = emc.make_workspace(cfg.n, n_pix, n_rot, n_pat)               # one workspace for the other stages
    w_ref, idx_ref = o.expand(inp.model_init, inp.q, quat[rows])
    assert np.array_equal(host(idx[t_rows]), idx_ref)
    w_s = host(w[t_rows])
    assert np.all(np.abs(w_s - w_ref) <= 1e-5 * np.abs(w_ref) + 1e-9 * np.abs(w_ref).max())

    # ---- stage 2 on the GPU's W (identical to the oracle's within 1e-5, checked above): sampled rows of L
    big_l = emc.emc_loglik(w, idx, d_q, d_mask, d_k, ws=ws)
    l_ref, a_ref = o.loglik(w_s, idx_ref, inp.counts, inp.mask)
    err = np.abs(host(big_l[t_rows]) - l_ref) / a_ref
    assert err.max() <= 1e-5, f"max |dL|/A = {err.max():.3e}"
    del w, idx
    torch.cuda.empty_cache()

    # ---- stage 3 stage-wise on sampled columns (each needs all R rows of the GPU's L)
    p, s, ll = emc.emc_normalize(big_l, d_quat, dev(weight), ws=ws)
    cols = np.unique(np.concatenate([np.random.default_rng(8).integers(0, n_pat, size=n_cols), [0, n_pat - 1]]))
    t_cols = torch.from_numpy(cols).cuda()
    p_ref, _, _ = o.normalize(host(big_l[:, t_cols]), weight)
    assert np.abs(host(p[:, t_cols]) - p_ref).max() <= 1e-6
    colsum = host(p.sum(dim=0, dtype=torch.float64))
    assert np.abs(colsum - 1).max() <= 1e-4
    s_ref = host(p.sum(dim=1, dtype=torch.float64))
    assert np.abs(host(s) - s_ref).max() <= 1e-5 * max(1.0, s_ref.max())

    # ---- stage 4 stage-wise on sampled rows: W'[r,:] = sum_d P[r,d] K[d,:] / s[r] from the GPU's P
    wn = emc.emc_update(p, s, d_q, d_mask, d_k, ws=ws)
    p_rows = host(p[t_rows])
    wn_ref, _ = o.update(p_rows, inp.counts, inp.mask)
    s_rows = p_rows.astype(np.float64).sum(axis=1)
    got = host(wn[t_rows])
    keep = s_rows > 1e-20
    scale = np.abs(wn_ref[keep]).max()
    rel = np.abs(got[keep] - wn_ref[keep]) / (np.abs(wn_ref[keep]) + 1e-7 * scale)
    assert rel.max() <= 2e-5, f"max rel dW' = {rel.max():.3e}"       # s[r] itself is a float32 sum on the GPU
    # photon conservation over ALL rows: sum_r s[r] W'[r,p] = sum_d K[d,p] on unmasked pixels
    tot = torch.zeros(n_pix, dtype=torch.float64, device="cuda")
    for r0 in range(0, n_rot, 2048):
        tot += (wn[r0:r0 + 2048].double() * s[r0:r0 + 2048].double()[:, None]).sum(dim=0)
    tot = host(tot)
    k_tot = inp.counts.astype(np.float64).sum(axis=0)
    use = inp.mask.astype(bool)
    assert np.abs(tot[use] - k_tot[use]).max() <= 1e-4 * max(1.0, k_tot[use].max())

    # ---- stage 5 over ALL rotations of the GPU's W' (the oracle scatters them in float64): the longest chains of float32
    # reductions per voxel that the config produces (T3, eq. 2.10; "division as a final step" :166)
    sw = (host(s) > 0).astype(np.float32)
    d_sw = dev(sw)
    m, den = emc.emc_compress(wn, d_sw, d_q, d_mask, d_quat, cfg.n, want_den=True, ws=ws)
    m_ref, den_ref = oracle_compress(host(wn), inp.q, quat, inp.mask, cfg.n, sw)
    m, den, m_ref = host(m).reshape(-1), host(den), m_ref.reshape(-1)
    cov = den_ref >= 1e-6 * den_ref.max()
    rel_den = np.abs(den[cov] - den_ref[cov]) / den_ref[cov]
    rel_m = np.abs(m[cov] - m_ref[cov]) / (np.abs(m_ref[cov]) + 1e-12)
    print(f"{name}: Compress over all {n_rot} rotations: max rel den {rel_den.max():.2e}, model {rel_m.max():.2e} "
          f"(most hits on a voxel {den_ref.max():.3g})")
    assert rel_den.max() <= 1e-5
    assert np.all(np.abs(m[cov] - m_ref[cov]) <= 1e-5 * np.abs(m_ref[cov]) + 1e-12), f"max rel {rel_m.max():.3e}"
    assert np.all(m[den_ref == 0] == 0)
    model_chain, ll_chain, s_chain = m, float(host(ll)[0]), host(s)
    del m_ref, den_ref

    # ---- the product path at this size: emc_iterate as bench.py times it (fused Expand with __logf planes, column
    # statistics from the contraction's epilogue, planes-only normalisation) against the oracle on the L it formed itself
    # and against the stage chain above (Algorithm 1)
    del p, wn, big_l
    torch.cuda.empty_cache()
    out = emc.emc_iterate(dev(inp.model_init), d_q, d_mask, d_quat, dev(weight), d_k, want_p=True, ws=ws)
    emc.emc_check(ws)
    torch.cuda.synchronize()
    l_it = emc.emc_workspace_view(ws, cfg.n, n_pix, n_rot, n_pat, emc.EMC_VIEW_LOGLIK)
    err = np.abs(host(l_it[t_rows]) - l_ref) / a_ref
    assert err.max() <= 1e-5, f"emc_iterate's own L: max |dL|/A = {err.max():.3e}"          # T1 on the product path's L
    p_ref, _, _ = o.normalize(host(l_it[:, t_cols]), weight)
    assert np.abs(host(out["P"][:, t_cols]) - p_ref).max() <= 1e-6                          # T2 on its P, stage-wise
    s_it = host(emc.emc_workspace_view(ws, cfg.n, n_pix, n_rot, n_pat, emc.EMC_VIEW_S))
    s_sum = host(out["P"].sum(dim=1, dtype=torch.float64))
    assert np.abs(s_it - s_sum).max() <= 1e-5 * max(1.0, s_sum.max())
    ll_it = float(host(out["loglik"])[0])
    assert abs(ll_it - ll_chain) <= 1e-6 * abs(ll_chain)
    # its W' rows from its own P (eq. 2.11), as for the stage call
    wn_it = host(emc.emc_workspace_view(ws, cfg.n, n_pix, n_rot, n_pat, emc.EMC_VIEW_WNEW)[t_rows])
    wn_ref2, _ = o.update(host(out["P"][t_rows]), inp.counts, inp.mask)
    keep = s_it[rows] > 1e-20
    scale = np.abs(wn_ref2[keep]).max()
    rel = np.abs(wn_it[keep] - wn_ref2[keep]) / (np.abs(wn_ref2[keep]) + 1e-7 * scale)
    assert rel.max() <= 2e-5, f"emc_iterate's own W': max rel {rel.max():.3e}"
    # model' of the two routes: the same arithmetic from L onwards, L itself differs by logf / __logf in the planes
    m_it = host(out["model"]).reshape(-1)
    big = np.abs(model_chain) >= 1e-6 * np.abs(model_chain).max()
    rel = np.abs(m_it - model_chain)[big] / np.abs(model_chain)[big]
    flips = int(((s_it > 0) != (s_chain > 0)).sum())
    print(f"{name}: emc_iterate vs stage chain: model' rel median {np.median(rel):.2e} max {rel.max():.2e}, "
          f"slices with s > 0 on one route only: {flips}")
    assert np.median(rel) <= 1e-5 and rel.max() <= 1e-2, (np.median(rel), rel.max())


def test_c3_full_config_sampled(inputs_cache):
    run_case(inputs_cache, "C3", n_pat=50000, stage=0, n_rows=24, n_cols=48)


def test_c4_route_pattern_chunks_from_host(inputs_cache):
    """Config 4's route at its own geometry and chunk size.  emc_iterate (chunks of 25 000 streamed from pinned host
    memory, numerators added up by TMA reduce-add, rows divided after the last chunk) is compared with the same
    iteration assembled from the stage calls chunk by chunk, and every stage of that chain is checked against the
    oracle on sampled rows / columns as in run_case (the oracle cannot form 10 000 x 60 000 x 15 808 in float64 in the
    time a test has)."""
    n_pat, chunk = 60000, 25000
    inp = inputs_cache("C4", n_pat=n_pat)
    cfg = inp.cfg
    quat, weight = inp.quat[0], inp.weight[0]
    n_rot, n_pix = quat.shape[0], cfg.n_pix
    d_model, d_q, d_mask, d_quat, d_w = dev(inp.model_init), dev(inp.q.reshape(cfg.n_det, cfg.n_det, 3)), dev(inp.mask), dev(quat), dev(weight)
    pinned = torch.from_numpy(inp.counts).pin_memory()
    out = emc.emc_iterate(d_model, d_q, d_mask, d_quat, d_w, pinned, n_pat_chunk=chunk, flags=emc.EMC_PATTERNS_ON_HOST)
    emc.emc_check(out["ws"])
    model_a, ll_a = host(out["model"]).reshape(-1), float(host(out["loglik"])[0])
    del out
    torch.cuda.empty_cache()

    rows = sampled_rows(n_rot, 16, 11)
    t_rows = torch.from_numpy(rows).cuda()
    w, idx = emc.emc_expand(d_model, d_q, d_quat)
    w_ref, idx_ref = o.expand(inp.model_init, inp.q, quat[rows])
    assert np.array_equal(host(idx[t_rows]), idx_ref)
    ws = emc.make_workspace(cfg.n, n_pix, n_rot, chunk)
    s = torch.zeros(n_rot, dtype=torch.float32, device="cuda")
    ll = torch.zeros(1, dtype=torch.float64, device="cuda")
    wnum = torch.zeros((n_rot, n_pix), dtype=torch.float32, device="cuda")
    p_rows = np.zeros((len(rows), n_pat), np.float32)
    rng = np.random.default_rng(12)
    for d0 in range(0, n_pat, chunk):
        d1 = min(n_pat, d0 + chunk)
        d_k = dev(inp.counts[d0:d1])
        big_l = emc.emc_loglik(w, idx, d_q, d_mask, d_k, ws=ws)
        l_ref, a_ref = o.loglik(host(w[t_rows]), idx_ref, inp.counts[d0:d1], inp.mask)
        assert (np.abs(host(big_l[t_rows]) - l_ref) / a_ref).max() <= 1e-5
        p, s, ll = emc.emc_normalize(big_l, d_quat, d_w, flags=emc.EMC_ACCUMULATE, s=s, loglik=ll, ws=ws)
        cols = np.unique(np.concatenate([rng.integers(0, d1 - d0, size=24), [0, d1 - d0 - 1]]))
        t_cols = torch.from_numpy(cols).cuda()
        p_ref, _, _ = o.normalize(host(big_l[:, t_cols]), weight)
        assert np.abs(host(p[:, t_cols]) - p_ref).max() <= 1e-6
        p_rows[:, d0:d1] = host(p[t_rows])
        emc.emc_update(p, None, d_q, d_mask, d_k, flags=emc.EMC_ACCUMULATE, wnew=wnum, ws=ws)
        del big_l, p, d_k
    # numerators over all chunks on sampled rows, then eq. (2.5)'s division (G9: after the last chunk)
    wn_ref, s_ref = o.update(p_rows, inp.counts, inp.mask)
    s_rows = host(s[t_rows]).astype(np.float64)
    assert np.abs(s_rows - s_ref).max() <= 1e-5 * max(1.0, s_ref.max())
    keep = s_ref > 1e-20
    got = host(wnum[t_rows]).astype(np.float64)[keep] / s_rows[keep, None]
    scale = np.abs(wn_ref[keep]).max()
    assert (np.abs(got - wn_ref[keep]) / (np.abs(wn_ref[keep]) + 1e-7 * scale)).max() <= 2e-5
    wn = wnum / torch.where(s > 0, s, torch.ones_like(s))[:, None]
    wn[s <= 0] = 0
    m_b, _ = emc.emc_compress(wn, s, d_q, d_mask, d_quat, cfg.n, ws=ws)
    model_b, ll_b = host(m_b).reshape(-1), float(host(ll)[0])
    # the two routes: same arithmetic up to the order of float32 sums
    assert abs(ll_a - ll_b) <= 1e-6 * abs(ll_b)
    big = np.abs(model_b) >= 1e-6 * np.abs(model_b).max()
    rel = np.abs(model_a - model_b)[big] / np.abs(model_b)[big]
    assert np.array_equal(model_a == 0, model_b == 0)
    assert np.median(rel) <= 1e-5 and rel.max() <= 1e-2, (np.median(rel), rel.max())
    # Compress against the oracle on the first 1000 rotations of that W'
    sub = slice(0, 1000)
    sw = (host(s[sub]) > 0).astype(np.float32)
    m, den = emc.emc_compress(wn[sub].contiguous(), dev(sw), d_q, d_mask, d_quat[sub].contiguous(), cfg.n, want_den=True, ws=ws)
    m_ref, _, den_ref = o.compress(host(wn[sub]), inp.q, quat[sub], inp.mask, cfg.n, slice_w=sw)
    m, m_ref = host(m).reshape(-1), m_ref.reshape(-1)
    cov = den_ref >= 1e-6 * den_ref.max()
    assert np.all(np.abs(m[cov] - m_ref[cov]) <= 1e-5 * np.abs(m_ref[cov]) + 1e-12)


def test_c5_last_stage_geometry_sampled(inputs_cache):
    run_case(inputs_cache, "C5", n_pat=20000 if FULL else 1024, stage=4, n_rows=12, n_cols=32)

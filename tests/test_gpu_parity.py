"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element, on the same
seeded inputs (`-m gpu`).  Tolerances are the ones north_star states, read as DESIGN.md §4 T1-T4:

  idx     bit-exact
  L       |dL| <= 1e-5 * A[r,d],  A = sum_p mask (K |logW| + W)
  P       |dP| <= 1e-6 stage-wise (both sides normalise the same float32 L); end to end
          |dP| <= 1e-6 + P_ref (exp(2 max_r |dL[r,d]|) - 1) with the dL MEASURED in the same test
  model'  |dm| <= 1e-5 * |m| on voxels with den >= 1e-6 max den, stage-wise (same W' in)
  W, W'   relative 1e-5 (not stated by north_star; same class as the model)
"""
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


def p_bound(p_ref, l_gpu, l_ref):
    """End-to-end bound on the responsibilities (T2).  With d[r] = L_gpu - L_ref in a column,
    P' = P e^d[r] / sum_r' P[r'] e^d[r'] lies within P e^(+-2 m), m = max_r |d[r]|: a rigorous bound from the
    log-likelihood difference actually measured, plus T2's 1e-6 for the normalisation itself."""
    m = np.abs(l_gpu.astype(np.float64) - l_ref.astype(np.float64)).max(axis=0)
    return 1e-6 + p_ref * np.expm1(2.0 * m)[None, :]


def gpu_loglik(case, model=None):
    """The float32 L of the STAGE calls for this case (emc_expand, then emc_loglik: W stored as float32, logW planes by
    logw_split_kernel with logf).  Not the arithmetic of emc_iterate, whose Expand forms the planes in registers with
    __logf and whose contraction also writes the column statistics: for that L see iterate_loglik()."""
    w, idx = emc.emc_expand(case.d_model if model is None else model, case.d_q, case.d_quat)
    return host(emc.emc_loglik(w, idx, case.d_q, case.d_mask, case.d_counts))


def iterate_loglik(out, n, n_pix, n_rot, n_pat, flags=0):
    """The float32 L that the emc_iterate call behind `out` itself formed (one pattern chunk, dense path), read from where
    it lies in that call's workspace (emc_workspace_view): the product path's own L, not a stage call's."""
    torch.cuda.synchronize()
    return host(emc.emc_workspace_view(out["ws"], n, n_pix, n_rot, n_pat, emc.EMC_VIEW_LOGLIK, flags))


class Case:
    """A workload on both sides: numpy for the oracle, CUDA tensors for libemc."""

    def __init__(self, inp, stage=0):
        self.inp, self.cfg = inp, inp.cfg
        self.quat, self.weight = inp.quat[stage], inp.weight[stage]
        self.d_model = dev(inp.model_init)
        nd = inp.cfg.n_det
        self.d_q = dev(inp.q.reshape(nd, nd, 3))   # row-major 2-D detector: emc_detector.row_len = n_det (4 x 8 pixel tiles)
        self.d_q_flat = dev(inp.q)                  # [P, 3]: row_len = 0, 32 consecutive pixels per warp
        self.d_mask = dev(inp.mask)
        self.d_quat = dev(self.quat)
        self.d_weight = dev(self.weight)
        self.d_counts = dev(inp.counts)


@pytest.fixture(scope="module", params=["T1", "T2", "T3", "C1"])
def case(request, inputs_cache):
    inp = inputs_cache(request.param)
    return Case(inp, stage=len(inp.quat) - 1)


@pytest.fixture(scope="module")
def ref(case):
    """The oracle's iteration on this case, stage by stage (float32 at the boundaries)."""
    inp = case.inp
    return o.iterate(inp.model_init, inp.q, inp.mask, case.quat, case.weight, inp.counts)


@pytest.mark.parametrize("use_ws,tiled", [(True, True), (True, False), (False, False)], ids=["blocked-tiles", "blocked-rows", "gather"])
def test_expand_index_map_bit_exact_and_slices(case, ref, use_ws, tiled):
    w, idx = emc.emc_expand(case.d_model, case.d_q if tiled else case.d_q_flat, case.d_quat, use_ws=use_ws)
    assert np.array_equal(host(idx), ref["idx"])                     # T4: bit-exact
    w = host(w)
    scale = np.abs(ref["W"]).max()
    assert np.abs(w - ref["W"]).max() <= 1e-5 * scale
    assert np.all(np.abs(w - ref["W"]) <= 1e-5 * np.abs(ref["W"]) + 1e-9 * scale)
    assert np.all(w[ref["idx"] < 0] == 0)


@pytest.mark.parametrize("flags", [0, emc.EMC_GEMM_1CTA, emc.EMC_DEBUG_SIMT], ids=["tcgen05-pair", "tcgen05-1cta", "simt"])
def test_loglik_within_1e5_of_A(case, ref, flags):
    inp = case.inp
    big_l, big_a = o.loglik(ref["W"], ref["idx"], inp.counts, inp.mask)
    got = host(emc.emc_loglik(dev(ref["W"]), dev(ref["idx"]), case.d_q, case.d_mask, case.d_counts, flags=flags))
    err = np.abs(got - big_l) / big_a
    assert err.max() <= 1e-5, f"max |dL|/A = {err.max():.3e}"


def test_normalize_stagewise_1e6(case, ref):
    l32 = ref["L"]
    p_ref, s_ref, ll_ref = o.normalize(l32, case.weight)
    big_l = torch.zeros((l32.shape[0], emc.ld_for(l32.shape[1])), dtype=torch.float32, device="cuda")
    big_l[:, : l32.shape[1]] = dev(l32)
    p, s, ll = emc.emc_normalize(big_l[:, : l32.shape[1]], case.d_quat, case.d_weight)
    p = host(p)
    assert np.abs(p - p_ref).max() <= 1e-6                           # T2 stage-wise
    assert np.abs(p.sum(axis=0) - 1).max() <= 1e-5
    assert np.abs(host(s) - s_ref).max() <= 1e-5 * max(1.0, s_ref.max())
    assert abs(float(host(ll)[0]) - ll_ref) <= 1e-6 * abs(ll_ref)
    # uniform prior passed as NULL gives the same numbers
    p2, _, _ = emc.emc_normalize(big_l[:, : l32.shape[1]], case.d_quat, None)
    if np.allclose(case.weight, case.weight[0]):
        assert np.abs(host(p2) - p_ref).max() <= 1e-6


@pytest.mark.parametrize("flags", [0, emc.EMC_GEMM_1CTA, emc.EMC_DEBUG_SIMT], ids=["tcgen05-pair", "tcgen05-1cta", "simt"])
def test_update_stagewise(case, ref, flags):
    inp = case.inp
    # emc_update takes P as libemc stores it: float32 subnormals count as 0 (EMC_P_MIN, include/emc.h; G20).  The oracle's
    # update is given the same array, so that the comparison is of eq. (2.11) itself on every row, fragile ones included
    p32 = gates.flushed(ref["P"])
    wn_ref, s_ref = o.update(p32, inp.counts, inp.mask)
    n_pat = p32.shape[1]
    p = torch.zeros((p32.shape[0], emc.ld_for(n_pat)), dtype=torch.float32, device="cuda")
    p[:, :n_pat] = dev(p32)
    s = dev(s_ref.astype(np.float32))
    wn = host(emc.emc_update(p[:, :n_pat], s, case.d_q, case.d_mask, case.d_counts, flags=flags))
    tol = 1e-5
    # rows with a vanishing s[r] divide two tiny numbers: compare the numerators there
    scale = np.abs(wn_ref).max()
    assert np.all(np.abs(wn - wn_ref) <= tol * np.abs(wn_ref) + 1e-7 * scale), \
        f"max rel {np.max(np.abs(wn - wn_ref) / (np.abs(wn_ref) + 1e-7 * scale)):.3e}"
    assert np.all(wn[:, inp.mask == 0] == 0)


@pytest.mark.parametrize("weighted", [False, True], ids=["eq2.10", "eq2.12"])
def test_compress_stagewise(case, ref, weighted):
    inp = case.inp
    n = case.cfg.n
    s32 = ref["s"].astype(np.float32)
    om = s32 if weighted else (s32 > 0).astype(np.float32)
    m_ref, _, den_ref = o.compress(ref["Wn"], inp.q, case.quat, inp.mask, n, slice_w=om)
    flags = emc.EMC_COMPRESS_WEIGHTED if weighted else 0
    m, den = emc.emc_compress(dev(ref["Wn"]), dev(s32), case.d_q, case.d_mask, case.d_quat, n, flags=flags,
                              want_den=True)
    m, den = host(m).reshape(-1), host(den)
    m_ref = m_ref.reshape(-1)
    cov = den_ref >= 1e-6 * den_ref.max()
    assert np.all(np.abs(den[cov] - den_ref[cov]) <= 1e-5 * den_ref[cov])
    assert np.all(np.abs(m[cov] - m_ref[cov]) <= 1e-5 * np.abs(m_ref[cov]) + 1e-12), \
        f"max rel {np.max(np.abs(m[cov] - m_ref[cov]) / (np.abs(m_ref[cov]) + 1e-12)):.3e}"   # T3
    assert np.all(m[den_ref == 0] == 0)


def model_gate(m, ref, weighted, case, quat=None, s_gpu=None, dl_max=0.0, label=""):
    """End-to-end gate on model' (tests/gates.py): T3's 1e-5 is held stage-wise
    (test_compress_stagewise); end to end the float32 rounding of L moves P by up to P (e^(2 dL) - 1) ~ 1e-5 ... 1e-3
    relative.  The oracle keeps P as the plain float32 cast; the slices whose weights hang on float32 subnormals (where
    libemc's flush-to-zero storage differs, G20) are identified on the oracle's P and gated by their footprint."""
    inp = case.inp
    gates.model_gate(m, ref, weighted, inp.q, case.quat if quat is None else quat, inp.mask, float(inp.counts.max()),
                     s_gpu=s_gpu, dl_max=dl_max, label=label or f"{inp.cfg.name} {'eq2.12' if weighted else 'eq2.10'}")


@pytest.mark.parametrize("uniform_null", [False, True], ids=["weights", "weights=NULL"])
@pytest.mark.parametrize("weighted", [False, True], ids=["eq2.10", "eq2.12"])
def test_iterate_end_to_end(case, weighted, uniform_null):
    """Whole iteration through emc_iterate.  weights=NULL is the header's documented default (w_r = 1/R) and takes
    the `uniform` branch of the fused column statistics and normalize_kernel<true>; the oracle gets w = 1/R."""
    inp = case.inp
    n_rot = case.quat.shape[0]
    weight = np.full(n_rot, 1.0 / n_rot, np.float32) if uniform_null else case.weight
    if not uniform_null and np.allclose(weight, weight[0]):
        # the configs' lists carry equal weights: make the explicit-weight case a non-uniform prior
        weight = np.random.default_rng(5).uniform(0.25, 2.0, size=n_rot).astype(np.float32)
        weight /= weight.sum()
    r = o.iterate(inp.model_init, inp.q, inp.mask, case.quat, weight, inp.counts, weighted=weighted)
    flags = emc.EMC_COMPRESS_WEIGHTED if weighted else 0
    out = emc.emc_iterate(case.d_model, case.d_q, case.d_mask, case.d_quat, None if uniform_null else dev(weight),
                          case.d_counts, flags=flags, want_p=True)
    emc.emc_check(out["ws"])
    # T1 on the L this very call formed (fused Expand with __logf planes, statistics in the contraction's epilogue)
    l_it = iterate_loglik(out, case.cfg.n, inp.q.shape[0], n_rot, inp.counts.shape[0], flags)
    l64, big_a = o.loglik(r["W"], r["idx"], inp.counts, inp.mask)
    err = np.abs(l_it.astype(np.float64) - l64) / big_a
    assert err.max() <= 1e-5, f"emc_iterate's own L: max |dL|/A = {err.max():.3e}"
    p = host(out["P"])
    bound = p_bound(r["P"], l_it, r["L"])                      # the bound on P from the dL of the same call
    assert np.all(np.abs(p - r["P"]) <= bound), f"max dP {np.abs(p - r['P']).max():.3e}"
    # the slices and weights that went into Compress, on the same footing as the stage tests
    s_it = host(emc.emc_workspace_view(out["ws"], case.cfg.n, inp.q.shape[0], n_rot, inp.counts.shape[0], emc.EMC_VIEW_S, flags))
    assert np.abs(s_it - p.sum(axis=1)).max() <= 1e-5 * max(1.0, float(s_it.max()))
    assert np.abs(p.sum(axis=0) - 1).max() <= 1e-5
    ll = float(host(out["loglik"])[0])
    assert abs(ll - r["LL"]) <= 1e-5 * abs(r["LL"])
    dl_max = float(np.abs(l_it.astype(np.float64) - r["L"].astype(np.float64)).max())
    model_gate(host(out["model"]), r, weighted, case, s_gpu=s_it, dl_max=dl_max)


def test_iterate_pattern_chunks_against_the_chunked_oracle(inputs_cache):
    """Config 4's route (pattern chunks, counts streamed from pinned host memory through the staging buffers,
    numerators added up by TMA reduce-add, rows divided after the last chunk) against oracle.iterate with the same
    chunks (G9), element by element; and two iterations, so that every staging-buffer hand-over is exercised."""
    inp = inputs_cache("T2")
    c = Case(inp, stage=1)
    pinned = torch.from_numpy(inp.counts.copy()).pin_memory()
    for weighted in (False, True):
        ref = o.iterate(inp.model_init, inp.q, inp.mask, c.quat, c.weight, inp.counts, n_pat_chunk=200, weighted=weighted)
        one = o.iterate(inp.model_init, inp.q, inp.mask, c.quat, c.weight, inp.counts, weighted=weighted)
        flags = emc.EMC_COMPRESS_WEIGHTED if weighted else 0
        for counts, f in ((c.d_counts, flags), (pinned, flags | emc.EMC_PATTERNS_ON_HOST)):
            out = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, counts, n_pat_chunk=200, flags=f)
            emc.emc_check(out["ws"])
            ll = float(host(out["loglik"])[0])
            assert abs(ll - ref["LL"]) <= 1e-5 * abs(ref["LL"])
            model_gate(host(out["model"]), ref, weighted, c)
        # the oracle's own chunked and unchunked runs agree (pinned on the CPU too); the GPU's as well
        assert np.abs(ref["model"] - one["model"]).max() <= 1e-5 * np.abs(one["model"]).max()
    m = inp.model_init
    lls = []
    for _ in range(2):
        ref2 = o.iterate(m, inp.q, inp.mask, c.quat, c.weight, inp.counts, n_pat_chunk=200)
        m = ref2["model"]
        lls.append(ref2["LL"])
    out = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, pinned, n_iter=2, n_pat_chunk=200,
                          flags=emc.EMC_PATTERNS_ON_HOST)
    got = host(out["loglik"])
    assert abs(got[0] - lls[0]) <= 1e-5 * abs(lls[0]) and abs(got[1] - lls[1]) <= 1e-4 * abs(lls[1])
    rel = np.abs(host(out["model"]) - m).reshape(-1) / (np.abs(m).reshape(-1) + 1e-6 * np.abs(m).max())
    assert np.median(rel[ref2["den"] >= 1e-3 * ref2["den"].max()]) <= 1e-3


def test_iterate_chunked_matches_single_chunk(inputs_cache):
    inp = inputs_cache("T2")
    c = Case(inp, stage=1)
    a = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, c.d_counts)
    b = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, c.d_counts, n_pat_chunk=200)
    ma, mb = host(a["model"]), host(b["model"])
    assert np.abs(ma - mb).max() <= 1e-4 * np.abs(ma).max()
    assert abs(float(host(a["loglik"])[0]) - float(host(b["loglik"])[0])) <= 1e-6 * abs(float(host(a["loglik"])[0]))
    # patterns streamed from pinned host memory
    pinned = torch.from_numpy(inp.counts.copy()).pin_memory()
    h = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, pinned, n_pat_chunk=200,
                        flags=emc.EMC_PATTERNS_ON_HOST)
    assert np.abs(host(h["model"]) - mb).max() <= 1e-5 * np.abs(mb).max()
    # two iterations x three chunks through the two staging buffers = the same as device-resident patterns
    b2 = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, c.d_counts, n_iter=2, n_pat_chunk=200)
    h2 = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, pinned, n_iter=2, n_pat_chunk=200,
                         flags=emc.EMC_PATTERNS_ON_HOST)
    assert np.abs(host(h2["model"]) - host(b2["model"])).max() <= 1e-5 * np.abs(host(b2["model"])).max()
    assert np.allclose(host(h2["loglik"]), host(b2["loglik"]), rtol=1e-6)   # fp32 atomics order the second iteration


def test_iterate_multi_iteration_matches_repeated_calls(inputs_cache):
    inp = inputs_cache("T1")
    c = Case(inp)
    a = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, c.d_counts, n_iter=3)
    m = c.d_model
    lls = []
    for _ in range(3):
        out = emc.emc_iterate(m, c.d_q, c.d_mask, c.d_quat, c.d_weight, c.d_counts)
        m = out["model"]
        lls.append(float(host(out["loglik"])[0]))
    assert np.abs(host(a["model"]) - host(m)).max() <= 1e-3 * np.abs(host(m)).max()
    assert np.allclose(host(a["loglik"]), lls, rtol=1e-6)
    # and against three iterations of the oracle: the log-likelihood of iteration n sees the model errors of n - 1
    mo, ref = inp.model_init, None
    for n in range(3):
        ref = o.iterate(mo, inp.q, inp.mask, c.quat, c.weight, inp.counts)
        mo = ref["model"]
        assert abs(lls[n] - ref["LL"]) <= (1e-5 if n == 0 else 1e-4) * abs(ref["LL"]), (n, lls[n], ref["LL"])
    cov = ref["den"] >= 1e-3 * ref["den"].max()
    rel = np.abs(host(a["model"]).reshape(-1) - mo.reshape(-1))[cov] / (np.abs(mo.reshape(-1)[cov]) + 1e-6 * np.abs(mo).max())
    assert np.median(rel) <= 1e-3, np.median(rel)


def test_count_range_is_reported(inputs_cache):
    inp = inputs_cache("T0")
    c = Case(inp)
    k = inp.counts.copy()
    k[3, 5] = 5000                              # > EMC_MAX_COUNT = 2048
    out = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, dev(k))
    assert torch.isnan(out["model"]).all() and torch.isnan(out["loglik"]).all()      # cannot be consumed unnoticed
    with pytest.raises(emc.EmcError) as e:
        emc.emc_check(out["ws"])
    assert e.value.status == emc.EMC_ERR_COUNT_RANGE
    w, idx = emc.emc_expand(c.d_model, c.d_q, c.d_quat)
    assert torch.isnan(emc.emc_loglik(w, idx, c.d_q, c.d_mask, dev(k))).all()
    # a huge count under the mask is ignored
    k = inp.counts.copy()
    mask = inp.mask.copy()
    mask[5] = 0
    k[:, 5] = 2 ** 31 - 1
    out = emc.emc_iterate(c.d_model, c.d_q, dev(mask), c.d_quat, c.d_weight, dev(k))
    emc.emc_check(out["ws"])


def test_degenerate_sizes(inputs_cache):
    """One rotation, one pattern, sizes far below one tile."""
    inp = inputs_cache("T0")
    c = Case(inp)
    out = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat[:1].contiguous(), None, c.d_counts[:1].contiguous(),
                          want_p=True)
    assert np.allclose(host(out["P"]), 1.0)
    r = o.iterate(inp.model_init, inp.q, inp.mask, c.quat[:1], np.ones(1, np.float32), inp.counts[:1])
    cov = r["den"] > 0
    assert np.allclose(host(out["model"]).reshape(-1)[cov], r["model"].reshape(-1)[cov], rtol=1e-4, atol=1e-7)


def test_host_patterns_pipelined_first_iteration(inputs_cache):
    """N >= 4096 host-resident patterns in one chunk: the first iteration runs on four sub-ranges (ragged last one)
    while the copies are in flight; results = the device-resident run up to summation order."""
    inp = inputs_cache("T1", n_pat=4200)
    c = Case(inp)
    pinned = torch.from_numpy(inp.counts.copy()).pin_memory()
    for n_iter in (1, 2):
        a = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, c.d_counts, n_iter=n_iter, want_p=True)
        h = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, pinned, n_iter=n_iter, want_p=True,
                            flags=emc.EMC_PATTERNS_ON_HOST)
        emc.emc_check(h["ws"])
        ma, mh = host(a["model"]), host(h["model"])
        assert np.abs(ma - mh).max() <= 1e-5 * np.abs(ma).max()
        assert np.allclose(host(a["loglik"]), host(h["loglik"]), rtol=1e-6)
        assert np.abs(host(a["P"]) - host(h["P"])).max() <= (1e-6 if n_iter == 1 else 1e-4)
    ref = o.iterate(inp.model_init, inp.q, inp.mask, c.quat, c.weight, inp.counts)
    h1 = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, pinned, want_p=True,
                         flags=emc.EMC_PATTERNS_ON_HOST)
    assert abs(float(host(h1["loglik"])[0]) - ref["LL"]) <= 1e-5 * abs(ref["LL"])


@pytest.mark.parametrize("name", ["T1", "C1"])
def test_den_reuse_across_iterations(inputs_cache, name):
    """Inside one emc_iterate call the iterations after the first reuse den (eq. 2.10) while the set of skipped
    slices is unchanged and re-accumulate it when it changes (decided on the device); repeated single-iteration
    calls always accumulate both.  The two must agree to the order of the float32 atomics."""
    inp = inputs_cache(name)
    c = Case(inp)
    a = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, c.d_counts, n_iter=4)
    m = c.d_model
    for _ in range(4):
        m = emc.emc_iterate(m, c.d_q, c.d_mask, c.d_quat, c.d_weight, c.d_counts)["model"]
    ma, mb = host(a["model"]).reshape(-1), host(m).reshape(-1)
    big = np.abs(mb) >= 1e-6 * np.abs(mb).max()
    rel = np.abs(ma - mb)[big] / np.abs(mb)[big]
    assert np.array_equal(ma == 0, mb == 0)                 # the same voxels are covered
    # run-to-run variation of four iterations is itself 1e-3 at the worst voxel (atomics order, amplified by peaked
    # responsibilities on C1) and 1.5e-6 in the median; a stale or double-counted den would move the median
    assert rel.max() <= 2e-2 and np.median(rel) <= 1e-5, (rel.max(), np.median(rel))
    # the oracle's four iterations (it accumulates den afresh every time)
    mo, ref = inp.model_init, None
    for _ in range(4):
        ref = o.iterate(mo, inp.q, inp.mask, c.quat, c.weight, inp.counts)
        mo = ref["model"]
    cov = ref["den"] >= 1e-3 * ref["den"].max()
    rel = np.abs(ma - mo.reshape(-1))[cov] / (np.abs(mo.reshape(-1)[cov]) + 1e-6 * np.abs(mo).max())
    assert np.median(rel) <= 1e-3, np.median(rel)
    assert np.array_equal(ma[ref["den"] == 0] == 0, np.ones(int((ref["den"] == 0).sum()), bool))


# ---------------------------------------------------------------------------------------------- rotation chunks (NEXT-2)

@pytest.mark.parametrize("name,chunk,weighted,null_w", [("T1", 64, False, False), ("T1", 100, True, True), ("T2", 128, True, False),
                                                        ("T2", 333, False, False), ("T3", 40, False, True), ("C1", 200, False, False)])
def test_iterate_rot_chunked_matches_oracle(inputs_cache, name, chunk, weighted, null_w):
    """emc_iterate_rot_chunked against the oracle's streamed iteration and against the GPU's own
    unchunked emc_iterate: LL, and model' on the covered voxels, for ragged last chunks, one chunk, NULL weights."""
    inp = inputs_cache(name)
    c = Case(inp, stage=len(inp.quat) - 1)
    n_rot = c.quat.shape[0]
    w = np.full(n_rot, 1.0 / n_rot, np.float32) if null_w else c.weight
    ref = o.iterate_rotation_chunks(inp.model_init, inp.q, inp.mask, c.quat, w, inp.counts, chunk, weighted=weighted)
    flags = emc.EMC_COMPRESS_WEIGHTED if weighted else 0
    out = emc.emc_iterate_rot_chunked(c.d_model, c.d_q, c.d_mask, c.d_quat, None if null_w else c.d_weight, c.d_counts, chunk,
                                      flags=flags)
    emc.emc_check(out["ws"])
    one = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, None if null_w else c.d_weight, c.d_counts, flags=flags)
    ll = float(host(out["loglik"])[0])
    assert abs(ll - ref["LL"]) <= 1e-5 * abs(ref["LL"])
    assert abs(ll - float(host(one["loglik"])[0])) <= 1e-6 * abs(ll)
    m, m1, m_ref = host(out["model"]).reshape(-1), host(one["model"]).reshape(-1), ref["model"].reshape(-1)
    cov = ref["den"] >= 1e-3 * ref["den"].max()
    scale = np.abs(m_ref).max()
    rel = np.abs(m - m_ref)[cov] / (np.abs(m_ref[cov]) + 1e-6 * scale)
    rel1 = np.abs(m - m1)[cov] / (np.abs(m1[cov]) + 1e-6 * scale)
    # end to end: the same gate as test_iterate_end_to_end (P amplifies the float32 rounding of L);
    # the fragile slices are read off the unchunked oracle's P (the same numbers: test_oracle_pins)
    full = o.iterate(inp.model_init, inp.q, inp.mask, c.quat, w, inp.counts, weighted=weighted)
    model_gate(m, dict(ref, P=full["P"], model=ref["model"]), weighted, c, label=f"{name} rotation chunks of {chunk}")
    assert np.median(rel1) <= 1e-5 and rel1.max() <= 2e-2, (np.median(rel1), rel1.max())
    assert np.array_equal(m == 0, m1 == 0)


def test_iterate_rot_chunked_two_iterations(inputs_cache):
    inp = inputs_cache("T1")
    c = Case(inp)
    a = emc.emc_iterate_rot_chunked(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, c.d_counts, 96, n_iter=2)
    b = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, c.d_counts, n_iter=2)
    assert np.allclose(host(a["loglik"]), host(b["loglik"]), rtol=2e-6)
    ma, mb = host(a["model"]).reshape(-1), host(b["model"]).reshape(-1)
    big = np.abs(mb) >= 1e-3 * np.abs(mb).max()
    assert np.median(np.abs(ma - mb)[big] / np.abs(mb)[big]) <= 1e-5


# ---------------------------------------------------------------------------------------------- photon lists (NEXT-2)

@pytest.mark.parametrize("name,chunk,weighted,n_iter", [("T1", 0, False, 1), ("T1", 50, True, 1), ("T2", 200, False, 2), ("T3", 0, True, 1),
                                                        ("C1", 0, False, 1), ("C1", 300, False, 2)])
def test_iterate_sparse_photons_matches_oracle(inputs_cache, name, chunk, weighted, n_iter):
    """EMC_SPARSE_PHOTONS: stages 2 and 4 from photon lists (emc_sparse.cu) against the oracle (whose photon-list forms are
    pinned to the dense definitions) with the end-to-end gates of test_iterate_end_to_end, and against the dense
    tensor-core path of the same library."""
    inp = inputs_cache(name)
    c = Case(inp, stage=len(inp.quat) - 1)
    flags = (emc.EMC_COMPRESS_WEIGHTED if weighted else 0)
    mo, ref = inp.model_init, None
    for _ in range(n_iter):
        ref = o.iterate(mo, inp.q, inp.mask, c.quat, c.weight, inp.counts, n_pat_chunk=chunk or None, weighted=weighted)
        mo = ref["model"]
    want_p = chunk == 0
    out = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, c.d_counts, n_iter=n_iter, n_pat_chunk=chunk,
                          flags=flags | emc.EMC_SPARSE_PHOTONS, want_p=want_p)
    emc.emc_check(out["ws"])
    dense = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, c.d_counts, n_iter=n_iter, n_pat_chunk=chunk,
                            flags=flags, want_p=want_p)
    ll = host(out["loglik"])
    assert abs(ll[-1] - ref["LL"]) <= (1e-5 if n_iter == 1 else 1e-4) * abs(ref["LL"])
    assert np.allclose(ll, host(dense["loglik"]), rtol=1e-5 if n_iter == 1 else 1e-4)   # LL is a sum of terms that largely cancel
    if want_p and n_iter == 1:
        l_gpu = gpu_loglik(c)
        p = host(out["P"])
        assert np.all(np.abs(p - ref["P"]) <= 2 * p_bound(ref["P"], l_gpu, ref["L"]))
        assert np.abs(p.sum(axis=0) - 1).max() <= 1e-5
    m, md, m_ref = host(out["model"]).reshape(-1), host(dense["model"]).reshape(-1), ref["model"].reshape(-1)
    cov = ref["den"] >= 1e-3 * ref["den"].max()
    scale = np.abs(m_ref).max()
    rel = np.abs(m - m_ref)[cov] / (np.abs(m_ref[cov]) + 1e-6 * scale)
    reld = np.abs(m - md)[cov] / (np.abs(md[cov]) + 1e-6 * scale)
    lim = (1e-4, 5e-2) if n_iter == 1 else (1e-3, 0.5)
    if n_iter == 1:
        model_gate(m, ref, weighted, c, label=f"{name} photon lists")
    else:       # the second iteration starts from models that already differ where a fragile slice (G20) took part or not
        assert np.median(rel) <= lim[0] and rel.max() <= lim[1], (np.median(rel), rel.max())
    assert np.median(reld) <= lim[0] and reld.max() <= lim[1], (np.median(reld), reld.max())
    # a voxel that is exactly 0 on one side (responsibilities below 2^-40 of their chunk's maximum vanish from the dense
    # path's fp16 operand planes) is at most a rounding error of the largest voxel on the other
    assert np.abs(m - md)[(m == 0) | (md == 0)].max(initial=0.0) <= 1e-7 * scale


def test_iterate_sparse_photons_host_patterns(inputs_cache):
    inp = inputs_cache("T2")
    c = Case(inp, stage=1)
    pinned = torch.from_numpy(inp.counts.copy()).pin_memory()
    a = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, pinned, n_pat_chunk=200,
                        flags=emc.EMC_SPARSE_PHOTONS | emc.EMC_PATTERNS_ON_HOST)
    b = emc.emc_iterate(c.d_model, c.d_q, c.d_mask, c.d_quat, c.d_weight, c.d_counts, n_pat_chunk=200, flags=emc.EMC_SPARSE_PHOTONS)
    emc.emc_check(a["ws"])
    assert np.allclose(host(a["loglik"]), host(b["loglik"]), rtol=1e-7)
    assert np.abs(host(a["model"]) - host(b["model"])).max() <= 1e-5 * np.abs(host(b["model"])).max()

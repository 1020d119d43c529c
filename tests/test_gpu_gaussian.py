"""Parity of emc_iterate_gaussian (the paper's Gaussian likelihood with fluence, eqs. 2.2-2.6; DESIGN.md section 11
NEXT-3) with the oracle, which evaluates eq. (2.2) term by term in float64.  (`-m gpu`)

Tolerances: Q is not exposed by the C ABI (the kernels carry B = sum_p W K), so the E-step is checked through
P: |dP| <= 1e-6 + 2 P_ref max_r |dQ| with |dQ| <= 1e-5 A[r,d], A = sum_p ((K/phi)^2 + W^2) / (2 sigma^2) (the scale
of the float32 terms Q is the difference of; same form as T1/T2 of the Poisson path); LL relative 1e-5 of the scale
sum_d max_r A; model' as in the Poisson end-to-end test."""
import numpy as np
import pytest
import torch

from oracle import emc_oracle as o

pytestmark = pytest.mark.gpu

emc = pytest.importorskip("paper_1409_4256_b200")


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


@pytest.mark.parametrize("name,sigma", [("T1", 20.0), ("T1", 5.0), ("T2", 10.0), ("C1", 30.0), ("T1null", 20.0)])
@pytest.mark.parametrize("weighted", [True, False], ids=["eq2.12", "eq2.10"])
def test_iterate_gaussian_matches_oracle(inputs_cache, name, sigma, weighted):
    null_weight = name.endswith("null")                      # weight = NULL: log(1/R) handed to both kernels by the host
    name = name.replace("null", "")
    inp = inputs_cache(name)
    stage = len(inp.quat) - 1
    quat, weight = inp.quat[stage], inp.weight[stage]
    if name == "T2":                                         # non-uniform prior weights
        rng = np.random.default_rng(3)
        weight = rng.uniform(0.5, 1.5, size=weight.shape).astype(np.float32)
        weight /= weight.sum()
    ref = o.iterate_gaussian(inp.model_init, inp.q, inp.mask, quat, weight, inp.counts, sigma, weighted=weighted)
    flags = emc.EMC_COMPRESS_WEIGHTED if weighted else 0
    out = emc.emc_iterate_gaussian(dev(inp.model_init), dev(inp.q), dev(inp.mask), dev(quat),
                                   None if null_weight else dev(weight), dev(inp.counts), sigma, flags=flags, want_p=True)
    emc.emc_check(out["ws"])
    p = out["P"].cpu().numpy()
    dq = 1e-5 * ref["A"].max(axis=0)                         # per column
    bound = 1e-6 + 2.0 * ref["P"] * dq[None, :]
    assert np.all(np.abs(p - ref["P"]) <= bound), f"max dP {np.abs(p - ref['P']).max():.3e}"
    assert np.abs(p.sum(axis=0) - 1).max() <= 1e-5
    ll = float(out["loglik"].cpu()[0])
    assert abs(ll - ref["LL"]) <= dq.sum(), (ll, ref["LL"])
    m, m_ref = out["model"].cpu().numpy().reshape(-1), ref["model"].reshape(-1)
    cov = ref["den"] >= 1e-3 * ref["den"].max()
    rel = np.abs(m[cov] - m_ref[cov]) / (np.abs(m_ref[cov]) + 1e-6 * np.abs(m_ref).max())
    assert np.median(rel) <= 1e-4 and rel.max() <= 5e-2, f"model rel: median {np.median(rel):.2e} max {rel.max():.2e}"


def test_gaussian_multi_iteration_and_arguments(inputs_cache):
    inp = inputs_cache("T1")
    args = (dev(inp.model_init), dev(inp.q), dev(inp.mask), dev(inp.quat[0]), dev(inp.weight[0]), dev(inp.counts))
    a = emc.emc_iterate_gaussian(*args, 10.0, n_iter=2)
    m = args[0]
    lls = []
    for _ in range(2):
        out = emc.emc_iterate_gaussian(m, *args[1:], 10.0)
        m = out["model"]
        lls.append(float(out["loglik"].cpu()[0]))
    assert np.allclose(a["loglik"].cpu().numpy(), lls, rtol=1e-6)
    with pytest.raises(emc.EmcError):
        emc.emc_iterate_gaussian(*args, 0.0)
    # host-resident patterns go through the staging buffers
    pinned = torch.from_numpy(inp.counts.copy()).pin_memory()
    h = emc.emc_iterate_gaussian(*args[:5], pinned, 10.0, n_iter=2, flags=emc.EMC_PATTERNS_ON_HOST)
    assert np.allclose(h["loglik"].cpu().numpy(), lls, rtol=1e-6)


@pytest.mark.parametrize("name,sigma", [("T1", 20.0), ("T2", 6.0), ("T3", 10.0), ("C1", 30.0)])
def test_loglik_gaussian_stage_q_and_phi(inputs_cache, name, sigma):
    """The E-step of the Gaussian model on its own (eqs. 2.2, 2.3, 2.6): the exponent Q against the oracle's term-by-term
    sum within 1e-5 of its scale A[r,d] = sum((K/phi)^2 + W^2) / (2 sigma^2) (the tolerance DESIGN.md section 11 states for the
    collapsed form), and the fluence phi to relative 1e-5."""
    inp = inputs_cache(name)
    stage = len(inp.quat) - 1
    w_ref, idx = o.expand(inp.model_init, inp.q, inp.quat[stage])
    phi_ref = o.fluence(w_ref, inp.counts, inp.mask)
    q_ref, a_ref = o.gaussian_loglik(w_ref, inp.counts, inp.mask, phi_ref, sigma)
    big_q, phi = emc.emc_loglik_gaussian(dev(w_ref), dev(inp.q), dev(inp.mask), dev(inp.counts), sigma)
    big_q, phi = big_q.cpu().numpy().astype(np.float64), phi.cpu().numpy().astype(np.float64)
    assert np.all(np.abs(big_q - q_ref) <= 1e-5 * a_ref + 1e-30), f"max dQ/A {np.max(np.abs(big_q - q_ref) / (a_ref + 1e-30)):.3e}"
    fin = np.isfinite(phi_ref)
    assert np.array_equal(np.isfinite(phi), fin)
    assert np.all(np.abs(phi[fin] - phi_ref[fin]) <= 1e-5 * np.abs(phi_ref[fin]))


@pytest.mark.parametrize("name,chunk", [("T1", 50), ("T2", 200)])
def test_iterate_gaussian_pattern_chunks(inputs_cache, name, chunk):
    """Pattern chunks of the Gaussian model: fluence and E-step are per frame, so the chunked run equals the one-chunk run
    (and through it the oracle) up to summation order; host-resident chunks go through the staging buffers."""
    inp = inputs_cache(name)
    stage = len(inp.quat) - 1
    args = (dev(inp.model_init), dev(inp.q), dev(inp.mask), dev(inp.quat[stage]), dev(inp.weight[stage]), dev(inp.counts))
    ref = o.iterate_gaussian(inp.model_init, inp.q, inp.mask, inp.quat[stage], inp.weight[stage], inp.counts, 15.0)
    one = emc.emc_iterate_gaussian(*args, 15.0, flags=emc.EMC_COMPRESS_WEIGHTED)
    pinned = torch.from_numpy(inp.counts.copy()).pin_memory()
    for counts, extra in ((args[5], 0), (pinned, emc.EMC_PATTERNS_ON_HOST)):
        out = emc.emc_iterate_gaussian(*args[:5], counts, 15.0, n_pat_chunk=chunk, flags=emc.EMC_COMPRESS_WEIGHTED | extra)
        emc.emc_check(out["ws"])
        ll, ll1 = float(out["loglik"].cpu()[0]), float(one["loglik"].cpu()[0])
        assert abs(ll - ll1) <= 1e-6 * abs(ll1) and abs(ll - ref["LL"]) <= 1e-5 * ref["A"].max(axis=0).sum()
        m, m1, m_ref = (x.reshape(-1) for x in (out["model"].cpu().numpy(), one["model"].cpu().numpy(), ref["model"]))
        cov = ref["den"] >= 1e-3 * ref["den"].max()
        scale = np.abs(m_ref).max()
        assert np.median(np.abs(m - m1)[cov] / (np.abs(m1[cov]) + 1e-6 * scale)) <= 1e-5
        rel = np.abs(m - m_ref)[cov] / (np.abs(m_ref[cov]) + 1e-6 * scale)
        assert np.median(rel) <= 1e-4 and rel.max() <= 5e-2


def test_gaussian_slice_range_is_reported(inputs_cache):
    """Slices at or above 65504 do not fit the fp16 planes of W: emc_check says so instead of letting inf / NaN pass."""
    inp = inputs_cache("T1")
    args = [dev(inp.model_init * np.float32(1e9 / inp.model_init.max())), dev(inp.q), dev(inp.mask), dev(inp.quat[0]),
            dev(inp.weight[0]), dev(inp.counts)]
    out = emc.emc_iterate_gaussian(*args, 10.0)
    with pytest.raises(emc.EmcError) as e:
        emc.emc_check(out["ws"])
    assert e.value.status == emc.EMC_ERR_VALUE_RANGE
    ok = emc.emc_iterate_gaussian(dev(inp.model_init), *args[1:], 10.0, ws=out["ws"])
    emc.emc_check(ok["ws"])                                   # the record is cleared by the check and by the next call

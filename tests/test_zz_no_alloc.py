"""emc_normalize_static: stage 3 for callers that cannot allocate device memory.

Some users of libemc get a fixed set of device buffers and nothing more: a plug-in inside an acquisition program, a
loop that has to stay clear of cudaMalloc's device-wide lock while frames stream in, a process whose pool is already
handed out.  They cannot build the workspace every other call wants.  For them the library carries one
EMC_STATIC_SCRATCH_BYTES array of its own (include/emc.h); the caller passes only L and the outputs.

What is checked here: the same numbers as emc_normalize (the workspace path the other tests pin to the oracle), at the
stage-wise tolerances of tests/test_gpu_parity.py, on two calls in a row whose sizes differ -- the second call finds the
first one's leftovers in the shared array and must not be disturbed by them -- and that a repeated call leaves the
device's free memory where it was.  Sizes beyond the built-in array are refused before anything is enqueued.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here should not hide the parity
tests.  It passes alone in a fresh process (the first call does the per-device set-up) and after the other tests.
"""
import numpy as np
import pytest
import torch

emc = pytest.importorskip("paper_1409_4256_b200")


def _case(seed, n_rot, n_pat, weighted):
    """A float32 log-likelihood matrix of the size class and spread of a T1-C1 E-step, rows ld_n apart."""
    rng = np.random.default_rng(seed)
    big_l = (-600.0 + 25.0 * rng.standard_normal((n_rot, n_pat))).astype(np.float32)
    weight = None
    if weighted:
        weight = rng.uniform(0.2, 1.0, n_rot)
        weight = (weight / weight.sum()).astype(np.float32)
    quat = np.zeros((n_rot, 4), dtype=np.float32)      # normalisation reads the weights only
    quat[:, 0] = 1.0
    return big_l, quat, weight


def _compare(big_l, quat, weight):
    n_rot, n_pat = big_l.shape
    ld = emc.ld_for(n_pat)
    d_l = torch.zeros((n_rot, ld), dtype=torch.float32, device="cuda")
    d_l[:, :n_pat] = torch.from_numpy(big_l).cuda()
    d_quat = torch.from_numpy(quat).cuda()
    d_w = None if weight is None else torch.from_numpy(weight).cuda()
    # the caller's buffers: inputs above, outputs here; nothing else exists for the call to use
    p_out = torch.full((n_rot, ld), float("nan"), dtype=torch.float32, device="cuda")
    s_out = torch.full((n_rot,), float("nan"), dtype=torch.float32, device="cuda")
    ll_out = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    emc.emc_normalize_static(d_l[:, :n_pat], d_quat, d_w, p_out[:, :n_pat], s_out, ll_out)
    # the existing path, scratch in a caller-made workspace
    p_ref, s_ref, ll_ref = emc.emc_normalize(d_l[:, :n_pat], d_quat, d_w)
    torch.cuda.synchronize()
    p, p_ref = p_out[:, :n_pat].cpu().numpy(), p_ref.cpu().numpy()
    s, s_ref = s_out.cpu().numpy(), s_ref.cpu().numpy()
    assert np.isfinite(p).all() and np.isfinite(s).all()
    assert np.abs(p - p_ref).max() <= 1e-6                                   # T2, stage-wise
    assert np.abs(p.sum(axis=0) - 1).max() <= 1e-5
    assert np.abs(s - s_ref).max() <= 1e-5 * max(1.0, float(s_ref.max()))
    ll, ll_ref = float(ll_out.cpu()[0]), float(ll_ref.cpu()[0])
    assert abs(ll - ll_ref) <= 1e-6 * abs(ll_ref)
    return d_l, d_quat, d_w, p_out, s_out, ll_out


@pytest.mark.gpu
def test_normalize_static_matches_workspace_path_twice_in_a_row():
    # call 1: several row splits, ragged column tail, non-uniform prior; fills a large part of the shared array
    _compare(*_case(11, 1500, 2000, True))
    # call 2, straight after: other sizes, uniform prior (NULL weights); the array still holds call 1's statistics
    keep = _compare(*_case(12, 333, 130, False))
    # a repeat of call 2 (all set-up and kernel loading behind us) must not move the device's free memory
    d_l, d_quat, d_w, p_out, s_out, ll_out = keep
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    emc.emc_normalize_static(d_l[:, :130], d_quat, d_w, p_out[:, :130], s_out, ll_out)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before
    # and back to the large case: the small call's leftovers sit at the start of the array now
    _compare(*_case(11, 1500, 2000, True))


def test_normalize_static_size_limit_is_stated_and_enforced():
    """No device needed: the size check comes before any CUDA call."""
    lib = emc.load()
    cap = emc.EMC_STATIC_SCRATCH_BYTES
    for n_rot in (1, 480, 25000, 400000):
        for n_pat in (1, 130, 1000, 10000, 25000, 50000, 100000):
            need = lib.emc_normalize_static_bytes(n_rot, n_pat, emc.ld_for(n_pat))
            assert 0 < need <= cap, (n_rot, n_pat, need)
    assert lib.emc_normalize_static_bytes(0, 10, 64) == 0
    assert lib.emc_normalize_static_bytes(10, 100, 64) == 0                  # ld_n < N
    n_pat = 200000
    assert lib.emc_normalize_static_bytes(1000, n_pat, emc.ld_for(n_pat)) > cap
    rot = emc.binding._Rotations(1000, 256, None)
    # aligned non-null stand-ins for L and P: the call must refuse before it looks at them
    rc = lib.emc_normalize_static(256, rot, n_pat, emc.ld_for(n_pat), 512, None, None, 0, None)
    assert rc == emc.EMC_ERR_STATIC_SCRATCH
    assert b"EMC_STATIC_SCRATCH_BYTES" in lib.emc_strerror(rc)
    assert lib.emc_normalize_static(None, rot, 10, 64, 512, None, None, 0, None) == emc.EMC_ERR_ARG

"""tcgen05 accumulates in fp32 with truncation (a same-sign sum drifts by about -1.07e-9 per K element);
the plane GEMM therefore carries long sums in round-to-nearest register accumulators over 512-element
chunks.  These tests hold the residual bias flat in K up to 65 536.  (`-m gpu`; `-s` prints
the numbers quoted in profiles/r01_accumulation_bias.md)"""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

emc = pytest.importorskip("paper_1409_4256_b200")


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


@pytest.mark.parametrize("n_pat", [1024, 16384, 65536])
def test_update_sum_bias_is_flat_in_k(n_pat):
    rng = np.random.Generator(np.random.PCG64(n_pat))
    n_rot, n_pix = 256, 384
    p = rng.random((n_rot, n_pat)).astype(np.float32)
    k = rng.poisson(0.5, (n_pat, n_pix)).astype(np.uint16)
    ref = p.astype(np.float64) @ k.astype(np.float64)
    pp = torch.zeros((n_rot, emc.ld_for(n_pat)), dtype=torch.float32, device="cuda")
    pp[:, :n_pat] = dev(p)
    q, mask = dev(np.zeros((n_pix, 3), np.float32)), dev(np.ones(n_pix, np.uint8))
    got = emc.emc_update(pp[:, :n_pat], None, q, mask, dev(k), flags=emc.EMC_UPDATE_RAW).cpu().numpy()
    rel = (got.astype(np.float64) - ref) / ref
    print(f"update K={n_pat:6d} fp16x2 scaled: mean signed rel {rel.mean():+.3e}  max |rel| {np.abs(rel).max():.3e}")
    assert abs(rel.mean()) <= 2e-6 and np.abs(rel).max() <= 4e-6


@pytest.mark.parametrize("n_pix", [4096, 65536])
def test_loglik_dot_bias_is_flat_in_k(n_pix):
    rng = np.random.Generator(np.random.PCG64(n_pix))
    n_rot, n_pat = 256, 256
    w = rng.uniform(0.01, 0.5, (n_rot, n_pix)).astype(np.float32)          # log W < 0 everywhere: same-sign sum
    k = rng.poisson(0.5, (n_pat, n_pix)).astype(np.uint16)
    ref = np.log(w.astype(np.float64)) @ k.astype(np.float64).T
    s = w.astype(np.float64).sum(axis=1)
    q, mask = dev(np.zeros((n_pix, 3), np.float32)), dev(np.ones(n_pix, np.uint8))
    got = emc.emc_loglik(dev(w), None, q, mask, dev(k)).cpu().numpy().astype(np.float64) + s[:, None]
    rel = (got - ref) / np.abs(ref)
    print(f"loglik K={n_pix:6d} fp16x2: mean signed rel {rel.mean():+.3e}  max |rel| {np.abs(rel).max():.3e}")
    assert abs(rel.mean()) <= 2e-6 and np.abs(rel).max() <= 4e-6


def test_fp16_subnormal_lo_plane_is_kept():
    """The lo plane of logW near 0 is an fp16 subnormal; the tensor core must not flush it."""
    n_rot, n_pix, n_pat = 64, 256, 64
    w = np.full((n_rot, n_pix), np.float32(1.0009766), np.float32)          # log W = 9.7609e-4: lo = 4.6e-9... subnormal
    w[:, ::2] = np.float32(0.99951172)
    k = np.full((n_pat, n_pix), 200, np.uint16)
    ref = np.log(w.astype(np.float64)) @ k.astype(np.float64).T
    s = w.astype(np.float64).sum(axis=1)
    q, mask = dev(np.zeros((n_pix, 3), np.float32)), dev(np.ones(n_pix, np.uint8))
    got = emc.emc_loglik(dev(w), None, q, mask, dev(k)).cpu().numpy().astype(np.float64) + s[:, None]
    a = np.abs(np.log(w.astype(np.float64))) @ k.astype(np.float64).T + s[:, None]
    assert np.abs(got - ref).max() <= 1e-5 * a.max()


def test_update_keeps_relative_precision_over_the_float32_range():
    """G20: responsibilities are kept down to float32's smallest normal number, 2^-126.  Rows whose values sit at
    2^-20, 2^-60, 2^-100 and 2^-125 (and one row that mixes all of them in one 512-pattern chunk) must come out
    of the update contraction with the same relative accuracy: the per-(row, chunk) scale of the fp16 planes is
    applied as two exact factors and its inverse may be a float32 subnormal."""
    rng = np.random.Generator(np.random.PCG64(99))
    n_rot, n_pat, n_pix = 40, 1500, 320
    p = rng.uniform(1.0, 2.0, (n_rot, n_pat))
    expo = np.array([-20, -60, -100, -125])
    p[:32] *= (2.0 ** expo)[np.arange(32) % 4][:, None]
    p[32:] *= 2.0 ** rng.choice(expo, size=(8, n_pat))
    p = p.astype(np.float32)
    assert p[p > 0].min() >= np.finfo(np.float32).tiny
    k = rng.poisson(0.7, (n_pat, n_pix)).astype(np.uint16)
    ref = p.astype(np.float64) @ k.astype(np.float64)
    pp = torch.zeros((n_rot, emc.ld_for(n_pat)), dtype=torch.float32, device="cuda")
    pp[:, :n_pat] = dev(p)
    q, mask = dev(np.zeros((n_pix, 3), np.float32)), dev(np.ones(n_pix, np.uint8))
    got = emc.emc_update(pp[:, :n_pat], None, q, mask, dev(k), flags=emc.EMC_UPDATE_RAW).cpu().numpy().astype(np.float64)
    # uniform rows: every term has the row's magnitude; mixed rows: relative to the largest term of the sum
    rel = np.abs(got - ref) / ref
    assert rel[:32].max() <= 4e-6, rel[:32].max()
    assert rel[32:].max() <= 4e-6, rel[32:].max()
    s = p.astype(np.float64).sum(axis=1).astype(np.float32)
    wn = emc.emc_update(pp[:, :n_pat], dev(s), q, mask, dev(k)).cpu().numpy().astype(np.float64)
    assert (np.abs(wn - ref / s[:, None].astype(np.float64)) / (ref / s[:, None])).max() <= 5e-6

"""Pins of the oracle's Gaussian-model functions (the paper's own likelihood, eqs. 2.2, 2.3, 2.5, 2.6, 2.11;
PAPER.md:70-89, 124-130; DESIGN.md section 11 NEXT-3): closed forms, brute-force loops on tiny inputs, algebraic
identities the formulas imply, and reduction to the Poisson-path routines where the two coincide."""
import numpy as np
import pytest

from emc_inputs import make_inputs
from oracle import emc_oracle as o


@pytest.fixture(scope="module")
def tiny():
    rng = np.random.default_rng(11)
    w = rng.uniform(0.1, 3.0, size=(7, 13)).astype(np.float32)
    k = rng.poisson(1.5, size=(5, 13)).astype(np.int32)
    mask = np.ones(13, dtype=np.uint8)
    mask[[2, 9]] = 0
    k[:, 2] = 10 ** 6                                     # garbage in masked pixels must never matter
    return w, k, mask


def test_fluence_closed_form_and_brute_force(tiny):
    w, k, mask = tiny
    # a frame that IS c times slice r has fluence c for that rotation: sum (cW)^2 / sum W cW = c
    frames = np.stack([2.5 * w[3].astype(np.float64), 0.25 * w[0].astype(np.float64)])
    phi = o.fluence(w, frames, None)
    assert abs(phi[3, 0] - 2.5) < 1e-12 and abs(phi[0, 1] - 0.25) < 1e-12
    phi = o.fluence(w, k, mask)
    for r in range(w.shape[0]):
        for d in range(k.shape[0]):
            num = sum(float(k[d, i]) ** 2 for i in range(13) if mask[i])
            den = sum(float(w[r, i]) * float(k[d, i]) for i in range(13) if mask[i])
            assert abs(phi[r, d] - num / den) <= 1e-12 * abs(num / den)
    # a frame with no photons: phi = inf, K / phi = 0
    assert np.all(np.isinf(o.fluence(w, np.zeros((1, 13)), mask)))


def test_gaussian_loglik_brute_force_and_identities(tiny):
    w, k, mask = tiny
    sigma = 0.7
    phi = o.fluence(w, k, mask)
    q, a = o.gaussian_loglik(w, k, mask, phi, sigma)
    use = mask.astype(bool)
    for r in range(w.shape[0]):
        for d in range(k.shape[0]):
            tot = 0.0
            for i in range(13):
                if mask[i]:
                    tot += -(float(k[d, i]) / phi[r, d] - float(w[r, i])) ** 2 / (2 * sigma ** 2)   # eq. (2.2)
            assert abs(q[r, d] - tot) <= 1e-12 * a[r, d]
    # with phi of eq. (2.6) the sum collapses to -(C_r - B_rd^2 / A_d) / (2 sigma^2)
    wd, kd = w.astype(np.float64)[:, use], k.astype(np.float64)[:, use]
    c = (wd ** 2).sum(axis=1)[:, None]
    b = wd @ kd.T
    ad = (kd ** 2).sum(axis=1)[None, :]
    assert np.allclose(q, -(c - b * b / ad) / (2 * sigma ** 2), rtol=1e-10, atol=1e-10)
    # sigma only scales: Q sigma^2 is constant
    q2, _ = o.gaussian_loglik(w, k, mask, phi, 2 * sigma)
    assert np.allclose(4 * q2, q, rtol=1e-12)
    # a frame that is exactly phi0 times a slice has Q = 0 at that rotation and Q < 0 elsewhere
    frames = (3.0 * w[2].astype(np.float64))[None, :]
    phi0 = o.fluence(w, frames, mask)
    qf, _ = o.gaussian_loglik(w, frames, mask, phi0, sigma)
    assert abs(qf[2, 0]) < 1e-12 and np.all(np.delete(qf[:, 0], 2) < -1e-6)
    # no photons: phi = inf and Q = -sum W^2 / (2 sigma^2)
    z = np.zeros((1, 13))
    qz, _ = o.gaussian_loglik(w, z, mask, o.fluence(w, z, mask), sigma)
    assert np.allclose(qz[:, 0], -c[:, 0] / (2 * sigma ** 2))


def test_update_gaussian(tiny):
    w, k, mask = tiny
    rng = np.random.default_rng(5)
    phi = o.fluence(w, k, mask)
    # one-hot responsibilities: the slice becomes the frame divided by its fluence (eq. 2.5)
    p = np.zeros((7, 5))
    p[4, 1] = 1.0
    wn, s = o.update_gaussian(p, k, mask, phi)
    use = mask.astype(bool)
    assert np.allclose(wn[4, use], k[1, use] / phi[4, 1], rtol=1e-6) and np.all(wn[4, ~use] == 0)
    assert np.all(wn[[0, 1, 2, 3, 5, 6]] == 0) and s[4] == 1.0
    # brute force
    p = rng.uniform(size=(7, 5))
    wn, s = o.update_gaussian(p, k, mask, phi)
    for r in range(7):
        for i in range(13):
            want = sum(p[r, d] * k[d, i] / phi[r, d] for d in range(5)) / p[r].sum() if mask[i] else 0.0
            assert abs(wn[r, i] - want) <= 1e-6 * max(1.0, abs(want))
    # phi == 1 is the Poisson-path update
    w1, _ = o.update(p, k, mask)
    w2, _ = o.update_gaussian(p, k, mask, np.ones_like(phi))
    assert np.array_equal(w1, w2)


def test_iterate_gaussian_recovers_orientations():
    inp = make_inputs("T1")
    out = o.iterate_gaussian(inp.model_true, inp.q, inp.mask, inp.quat[0], inp.weight[0], inp.counts, sigma=1.0)
    assert np.abs(out["P"].sum(axis=0) - 1).max() < 1e-5
    hit = (out["P"].argmax(axis=0) == inp.r_true).mean()
    # Poisson frames at 0.5 photons per pixel under a Gaussian model with a free fluence: far above the chance
    # level 1/203, well below the Poisson model's 97 % on the same data
    assert hit >= 0.2, hit
    assert np.isfinite(out["LL"]) and np.all(out["Wn"] >= 0)

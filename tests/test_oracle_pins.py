"""Pins for the CPU oracle (`-m "not gpu"`): closed forms, invariants, brute force on tiny inputs and
independent library routines.  Nothing here calls the CUDA path.  The pin table is DESIGN.md §5;
each test names the passage of PAPER.md / reading of DESIGN.md §3 it holds the oracle to.
"""
import itertools
import pathlib

import numpy as np
import pytest
import scipy.special
import scipy.stats
from scipy.ndimage import map_coordinates
from scipy.spatial.transform import Rotation

from emc_inputs import make_inputs, random_rotations, rotation_ladder, detector_geometry
from oracle import emc_oracle as o

GOLDEN = pathlib.Path(__file__).parent / "golden"


def rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


# ------------------------------------------------------------------ golden: eq. (2.7)

def test_rotation_ladder_matches_printed_values():
    """PAPER.md:95-98 prints M_rot(d) for d = 5,6,8,10,12 (the only printed numbers that touch the
    inputs of the path: the sizes of the rotation lists)."""
    rows = [l.split() for l in (GOLDEN / "eq_2_7_rotation_ladder.txt").read_text().splitlines()
            if l.strip() and not l.startswith("#")]
    d = np.array([int(r[0]) for r in rows])
    m = np.array([int(r[1]) for r in rows])
    assert np.array_equal(rotation_ladder(d), m)


# ------------------------------------------------------------------ rotation

def _quat_mul(a, b):
    w1, x1, y1, z1 = a
    w2, x2, y2, z2 = b
    return np.array([w1 * w2 - x1 * x2 - y1 * y2 - z1 * z2,
                     w1 * x2 + x1 * w2 + y1 * z2 - z1 * y2,
                     w1 * y2 - x1 * z2 + y1 * w2 + z1 * x2,
                     w1 * z2 + x1 * y2 - y1 * x2 + z1 * w2])


def test_rotation_matrix_orthonormal_det_identity():
    quat = random_rotations(200, 7)
    m = o.rotation_matrix(quat).astype(np.float64)
    eye = np.einsum("rab,rcb->rac", m, m)
    assert np.abs(eye - np.eye(3)).max() < 5e-7
    assert np.abs(np.linalg.det(m) - 1.0).max() < 5e-7
    assert np.array_equal(o.rotation_matrix(np.array([[1, 0, 0, 0]], np.float32))[0], np.eye(3, dtype=np.float32))


def test_rotation_matrix_equals_quaternion_sandwich_and_scipy():
    """R v = q (0,v) q*  computed independently, and scipy's Rotation (scalar-last)."""
    quat = random_rotations(50, 8)
    m = o.rotation_matrix(quat).astype(np.float64)
    v = rng(9).standard_normal((50, 3))
    for r in range(50):
        qd = quat[r].astype(np.float64)
        conj = qd * np.array([1, -1, -1, -1])
        sand = _quat_mul(_quat_mul(qd, np.concatenate([[0.0], v[r]])), conj)[1:]
        assert np.allclose(m[r] @ v[r], sand, atol=1e-6)
    ref = Rotation.from_quat(quat.astype(np.float64)[:, [1, 2, 3, 0]]).as_matrix()
    assert np.abs(m - ref).max() < 5e-7


def test_rotation_90_degrees_about_z_is_active():
    """Active convention: +90 deg about z takes x to y."""
    h = np.sqrt(0.5)
    m = o.rotation_matrix(np.array([[h, 0, 0, h]], np.float32))[0]
    assert np.allclose(m @ np.array([1, 0, 0]), [0, 1, 0], atol=1e-6)


# ------------------------------------------------------------------ coordinates / index map

def test_sample_coords_is_unfused_float32_sequence():
    """G4: x_a = ((R_a0 q_x + R_a1 q_y) + R_a2 q_z) + c with every op rounded to float32 -- checked
    against scalar numpy.float32 arithmetic written out element by element."""
    quat = random_rotations(5, 10)
    q = detector_geometry(6, 16)
    x = o.sample_coords(quat, q, 16)
    rm = o.rotation_matrix(quat)
    c = np.float32(8.0)
    for r, p, a in itertools.product(range(5), range(0, 36, 7), range(3)):
        t0 = np.float32(rm[r, a, 0] * q[p, 0])
        t1 = np.float32(rm[r, a, 1] * q[p, 1])
        t2 = np.float32(rm[r, a, 2] * q[p, 2])
        ref = np.float32(np.float32(np.float32(t0 + t1) + t2) + c)
        assert x[r, p, a] == ref
    assert x.dtype == np.float32


def test_index_map_identity_rotation_integer_q():
    n = 8
    pts = np.array([[0, 0, 0], [1, -2, 3], [-4, -4, -4], [3, 3, 3], [2, 0, -1]], np.float32)
    idx = o.index_map(np.array([[1, 0, 0, 0]], np.float32), pts, n)[0]
    exp = []
    for (x, y, z) in pts.astype(int):
        bx, by, bz = x + 4, y + 4, z + 4
        ok = all(0 <= b <= n - 2 for b in (bx, by, bz))
        exp.append((bx * n + by) * n + bz if ok else -1)
    assert list(idx) == exp
    assert idx[3] == -1                 # 3 + 4 = 7 = n-1: the +1 neighbour is outside (G7)


def test_index_map_outside_grid_is_minus_one():
    n = 8
    pts = np.array([[5.5, 0, 0], [-4.5, 0, 0], [0, 0, 3.2], [0, 0, 2.9]], np.float32)
    idx = o.index_map(np.array([[1, 0, 0, 0]], np.float32), pts, n)[0]
    assert list(idx[:3]) == [-1, -1, -1] and idx[3] == (4 * n + 4) * n + 6


# ------------------------------------------------------------------ Expand, eq. (2.9)

def test_expand_reproduces_affine_field_exactly():
    """Trilinear interpolation is exact on affine fields: model(x) = a + b.x  =>  W[r,p] =
    a + b.(R_r q_p + c).  Pins rotation convention, origin c = n/2 and axis order (z fastest)."""
    n = 12
    a, b = 0.7, np.array([0.3, -0.2, 0.11])
    g = np.arange(n, dtype=np.float64)
    model = (a + b[0] * g[:, None, None] + b[1] * g[None, :, None] + b[2] * g[None, None, :]).astype(np.float32)
    quat = random_rotations(40, 11)
    q = detector_geometry(10, n)
    w, idx = o.expand(model, q, quat)
    x = np.einsum("rab,pb->rpa", Rotation.from_quat(quat.astype(np.float64)[:, [1, 2, 3, 0]]).as_matrix(),
                  q.astype(np.float64)) + n / 2
    ref = a + x @ b
    assert (idx >= 0).all()
    assert np.abs(w - ref).max() < 2e-5      # float32 coordinates: |b| * ulp(x) ~ 1e-6


def test_expand_constant_model_and_single_voxel():
    n = 10
    quat = random_rotations(20, 12)
    q = detector_geometry(8, n)
    w, _ = o.expand(np.full((n, n, n), 3.25, np.float32), q, quat)
    assert np.abs(w - 3.25).max() < 1e-6
    model = rng(13).random((n, n, n)).astype(np.float32)
    pts = np.array([[1, 2, -3], [0, 0, 0]], np.float32)
    w, idx = o.expand(model, pts, np.array([[1, 0, 0, 0]], np.float32))
    assert w[0, 0] == model[6, 7, 2] and w[0, 1] == model[5, 5, 5]
    assert idx[0, 0] == (6 * n + 7) * n + 2


def test_expand_brute_force_over_all_voxels():
    """Eq. (2.9) literally: sum over ALL grid points l of f(p_l - x) model[l] with the tent-product
    kernel f(u) = prod_a max(0, 1 - |u_a|)."""
    n = 6
    model = rng(14).random((n, n, n)).astype(np.float32)
    quat = random_rotations(7, 15)
    q = (rng(16).random((9, 3)).astype(np.float32) - 0.5) * 3.0
    w, idx = o.expand(model, q, quat)
    x = o.sample_coords(quat, q, n).astype(np.float64)
    g = np.arange(n, dtype=np.float64)
    n_in = 0
    for r in range(7):
        for p in range(9):
            fx = np.maximum(0, 1 - np.abs(g - x[r, p, 0]))
            fy = np.maximum(0, 1 - np.abs(g - x[r, p, 1]))
            fz = np.maximum(0, 1 - np.abs(g - x[r, p, 2]))
            ref = np.einsum("i,j,k,ijk->", fx, fy, fz, model.astype(np.float64))
            if idx[r, p] < 0:
                assert w[r, p] == 0          # G7
            else:
                n_in += 1
                assert abs(w[r, p] - ref) < 1e-6
    assert n_in > 40


def test_expand_matches_scipy_map_coordinates():
    inp = make_inputs("T1")
    w, idx = o.expand(inp.model_true, inp.q, inp.quat[0])
    x = o.sample_coords(inp.quat[0], inp.q, inp.cfg.n).astype(np.float64)
    ref = map_coordinates(inp.model_true.astype(np.float64), x.reshape(-1, 3).T, order=1).reshape(w.shape)
    ok = idx >= 0
    assert ok.mean() > 0.99
    scale = np.abs(ref[ok]).max()
    assert np.abs(w[ok] - ref[ok]).max() < 1e-6 * scale


# ------------------------------------------------------------------ log-likelihood (north_star 2)

def test_loglik_equals_poisson_logpmf_up_to_constant():
    """sum_p log Poisson(K; W) = L - sum_p log K!   (the dropped term is constant in r)."""
    g = rng(20)
    w = g.uniform(0.05, 3.0, (6, 50)).astype(np.float32)
    k = g.poisson(1.0, (8, 50)).astype(np.int32)
    mask = (g.random(50) > 0.2).astype(np.uint8)
    big_l, big_a = o.loglik(w, np.zeros_like(w, dtype=np.int32), k, mask)
    use = mask.astype(bool)
    for r in range(6):
        for d in range(8):
            ref = scipy.stats.poisson.logpmf(k[d, use], w[r, use].astype(np.float64)).sum()
            ref += scipy.special.gammaln(k[d, use] + 1.0).sum()
            assert abs(big_l[r, d] - ref) < 1e-9 * big_a[r, d]


def test_loglik_brute_force_with_masked_garbage_floor_and_invalid():
    g = rng(21)
    w = g.uniform(0.0, 2.0, (4, 12)).astype(np.float32)
    w[0, 3] = 0.0                           # floor: log(1e-30)   (G8)
    idx = np.zeros((4, 12), np.int32)
    idx[1, 5] = -1
    w[1, 5] = 0.0                           # outside the grid: drops out of the sum (G7)
    k = g.poisson(1.0, (5, 12)).astype(np.int64)
    mask = np.ones(12, np.uint8)
    mask[[2, 7]] = 0
    k[:, [2, 7]] = 10 ** 6                  # garbage in masked pixels must be ignored (G16)
    big_l, big_a = o.loglik(w, idx, k, mask)
    for r in range(4):
        for d in range(5):
            tot = 0.0
            tot_a = 0.0
            for p in range(12):
                if not mask[p]:
                    continue
                lw = 0.0 if idx[r, p] < 0 else float(np.log(np.float64(max(w[r, p], np.float32(1e-30)))))
                tot += k[d, p] * lw - float(w[r, p])
                tot_a += k[d, p] * abs(lw) + float(w[r, p])
            assert abs(big_l[r, d] - tot) < 1e-9 * max(1.0, tot_a)
            assert abs(big_a[r, d] - tot_a) < 1e-9 * max(1.0, tot_a)


# ------------------------------------------------------------------ normalise (eq. 2.4 reconstructed)

def test_normalize_sums_to_one_and_matches_scipy_softmax():
    g = rng(30)
    big_l = (g.standard_normal((40, 17)) * 300 - 2000).astype(np.float32)
    wgt = g.random(40)
    wgt = (wgt / wgt.sum()).astype(np.float32)
    p, s, ll = o.normalize(big_l, wgt)
    assert np.abs(p.sum(axis=0) - 1).max() < 1e-12
    a = big_l.astype(np.float64) + np.log(wgt.astype(np.float64))[:, None]
    assert np.abs(p - scipy.special.softmax(a, axis=0)).max() < 1e-12
    assert abs(ll - scipy.special.logsumexp(a, axis=0).sum()) < 1e-9 * abs(ll)
    assert np.allclose(s, p.sum(axis=1))
    # shifting a column by a constant changes nothing but LL
    shift = g.standard_normal(17) * 50
    p2, _, ll2 = o.normalize(big_l.astype(np.float64) + shift[None, :], wgt)
    assert np.abs(p - p2).max() < 1e-10
    assert abs((ll2 - ll) - shift.sum()) < 1e-6


def test_normalize_is_prior_for_equal_likelihoods_and_definition_without_max():
    g = rng(31)
    wgt = g.random(9)
    wgt = (wgt / wgt.sum()).astype(np.float32)
    p, _, _ = o.normalize(np.full((9, 4), -123.0, np.float32), wgt)
    w64 = wgt.astype(np.float64)
    assert np.abs(p - (w64 / w64.sum())[:, None]).max() < 1e-15
    # small |L|: the plain definition w T / sum w T needs no max-subtraction
    big_l = g.standard_normal((9, 4)).astype(np.float32)
    t = wgt.astype(np.float64)[:, None] * np.exp(big_l.astype(np.float64))
    assert np.abs(o.normalize(big_l, wgt)[0] - t / t.sum(axis=0)).max() < 1e-14


def test_constant_model_gives_prior_responsibilities():
    """north_star invariant, exact form (DESIGN.md §4 T3'): a constant model makes every slice equal,
    so P[r,d] = w[r]."""
    inp = make_inputs("T0")
    wgt = rng(32).random(inp.cfg.n_rot[0])
    wgt = (wgt / wgt.sum()).astype(np.float32)
    out = o.iterate(np.full_like(inp.model_true, 0.8), inp.q, inp.mask, inp.quat[0], wgt, inp.counts)
    assert np.abs(out["P"] - wgt[:, None]).max() < 1e-6


# ------------------------------------------------------------------ update (eq. 2.5 / 2.11)

def test_update_one_hot_is_mean_of_assigned_patterns():
    g = rng(40)
    k = g.poisson(2.0, (30, 20)).astype(np.uint16)
    mask = np.ones(20, np.uint8)
    mask[4] = 0
    k[:, 4] = 65535
    assign = g.integers(0, 5, 30)
    p = np.zeros((6, 30), np.float32)
    p[assign, np.arange(30)] = 1.0          # rotation 5 gets nothing
    wn, s = o.update(p, k, mask)
    for r in range(5):
        ref = k[assign == r].astype(np.float64).mean(axis=0)
        ref[4] = 0
        assert np.abs(wn[r] - ref).max() < 1e-6
    assert (wn[5] == 0).all() and s[5] == 0      # G17
    assert (wn[:, 4] == 0).all()                  # G16


def test_update_conserves_photons_and_matches_loops():
    """sum_r s[r] W'[r,p] = sum_d K[d,p] for every unmasked pixel when sum_r P[r,d] = 1."""
    g = rng(41)
    k = g.poisson(0.7, (25, 15)).astype(np.int32)
    p = g.random((8, 25))
    p = (p / p.sum(axis=0)).astype(np.float32)
    wn, s = o.update(p, k, None)
    tot = (s[:, None] * wn.astype(np.float64)).sum(axis=0)
    assert np.abs(tot - k.sum(axis=0)).max() < 1e-4
    for r in range(8):
        for px in range(15):
            num = sum(float(p[r, d]) * float(k[d, px]) for d in range(25))
            den = sum(float(p[r, d]) for d in range(25))
            assert abs(wn[r, px] - num / den) < 1e-6


# ------------------------------------------------------------------ Compress (eq. 2.10 / 2.12)

def _scatter(v, q, quat, mask, n, slice_w=None):
    return o.compress(v, q, quat, mask, n, slice_w=slice_w)


def test_compress_is_adjoint_of_expand():
    """<Expand(M), V> = <M, Scatter(V)> with Scatter = the numerator of eq. (2.10): pins the
    weights and indices of Compress against Expand.  And Scatter(1) = the denominator."""
    n = 10
    g = rng(50)
    quat = random_rotations(30, 51)
    q = detector_geometry(9, n)
    model = g.random((n, n, n)).astype(np.float32)
    v = g.random((30, 81)).astype(np.float32)
    w, _ = o.expand(model, q, quat)
    _, num, den = _scatter(v, q, quat, None, n)
    lhs = (w.astype(np.float64) * v).sum()
    rhs = (model.reshape(-1).astype(np.float64) * num).sum()
    assert abs(lhs - rhs) < 1e-6 * abs(lhs)
    _, num1, den1 = _scatter(np.ones((30, 81), np.float32), q, quat, None, n)
    assert np.abs(num1 - den1).max() < 1e-12 and np.abs(den - den1).max() < 1e-12


def test_compress_constant_slices_give_constant_model_where_covered():
    n = 10
    quat = random_rotations(25, 52)
    q = detector_geometry(9, n)
    mask = np.ones(81, np.uint8)
    mask[40] = 0
    model, _, den = _scatter(np.full((25, 81), 2.5, np.float32), q, quat, mask, n)
    cov = den > 0
    assert cov.sum() > 100
    assert np.abs(model.reshape(-1)[cov] - 2.5).max() < 1e-6
    assert (model.reshape(-1)[~cov] == 0).all()


def test_compress_brute_force_and_weighted_form():
    """Eq. (2.10) and eq. (2.12) literally, looping over all voxels with the tent-product kernel."""
    n = 6
    g = rng(53)
    quat = random_rotations(5, 54)
    q = (g.random((7, 3)).astype(np.float32) - 0.5) * 3.5
    mask = np.array([1, 1, 0, 1, 1, 1, 1], np.uint8)
    wn = g.random((5, 7)).astype(np.float32)
    s = np.array([0.5, 0.0, 2.0, 1.0, 0.25], np.float32)
    x = o.sample_coords(quat, q, n).astype(np.float64)
    grid = np.arange(n, dtype=np.float64)
    valid = o.index_map(quat, q, n) >= 0
    for weighted in (False, True):
        om = s.astype(np.float64) if weighted else (s > 0).astype(np.float64)
        num = np.zeros((n, n, n))
        den = np.zeros((n, n, n))
        for r in range(5):
            for p in range(7):
                if not mask[p] or not valid[r, p] or om[r] == 0:
                    continue
                f = np.einsum("i,j,k->ijk", *[np.maximum(0, 1 - np.abs(grid - x[r, p, a])) for a in range(3)])
                num += f * om[r] * float(wn[r, p])
                den += f * om[r]
        ref = np.where(den > 0, num / np.where(den > 0, den, 1), 0)
        model, _, den_o = _scatter(wn, q, quat, mask, n, slice_w=om.astype(np.float32))
        assert np.abs(den_o.reshape(n, n, n) - den).max() < 1e-12
        assert np.abs(model - ref).max() < 1e-6


def test_eq_2_12_equals_eq_2_10_with_slice_weights():
    """G6: eq. (2.12) on un-normalised slices (eq. 2.11) == eq. (2.10) with om_r = s[r] on
    normalised slices.  Checked by evaluating (2.12) from its own definition."""
    n = 8
    g = rng(55)
    quat = random_rotations(12, 56)
    q = detector_geometry(7, n)
    k = g.poisson(1.0, (20, 49)).astype(np.int32)
    p = g.random((12, 20))
    p = (p / p.sum(axis=0)).astype(np.float32)
    wn, s = o.update(p, k, None)
    unnorm = p.astype(np.float64) @ k.astype(np.float64)            # eq. (2.11)
    _, num, _ = _scatter(unnorm.astype(np.float32), q, quat, None, n)
    _, den, _ = _scatter(np.broadcast_to(s[:, None], unnorm.shape).astype(np.float32), q, quat, None, n)
    ref = np.where(den > 0, num / np.where(den > 0, den, 1), 0)     # eq. (2.12)
    model, _, _ = _scatter(wn, q, quat, None, n, slice_w=s.astype(np.float32))
    cov = den > 0
    assert np.abs(model.reshape(-1)[cov] - ref[cov]).max() < 1e-5 * np.abs(ref[cov]).max()


# ------------------------------------------------------------------ iteration (Algorithm 1)

def test_expand_compress_round_trip_recovers_model_loosely():
    """north_star invariant in its honest form (DESIGN.md §4 T4'): Expand -> Compress smooths
    (eq. 2.10 is inverse-distance weighting), so recovery is approximate; exact for a
    constant model (tested above)."""
    inp = make_inputs("T2")
    quat = inp.quat[1]
    n = inp.cfg.n
    g = np.arange(n, dtype=np.float64) - n / 2
    smooth = np.exp(-(g[:, None, None] ** 2 + g[None, :, None] ** 2 + g[None, None, :] ** 2) / (2 * 6.0 ** 2))
    smooth = smooth.astype(np.float32)           # varies slowly on the voxel scale
    w, _ = o.expand(smooth, inp.q, quat)
    model, _, den = o.compress(w, inp.q, quat, inp.mask, n)
    cov = den.reshape(model.shape) > 0.5 * np.median(den[den > 0])
    err = np.linalg.norm((model - smooth)[cov]) / np.linalg.norm(smooth[cov])
    assert cov.sum() > 5000 and err < 0.05


def test_iterate_recovers_orientations_and_chunks_agree():
    inp = make_inputs("T2")
    a = o.iterate(inp.model_true, inp.q, inp.mask, inp.quat[1], inp.weight[1], inp.counts)
    assert (a["P"].argmax(axis=0) == inp.r_true).mean() > 0.7
    assert np.abs(a["P"].sum(axis=0) - 1).max() < 1e-5
    b = o.iterate(inp.model_true, inp.q, inp.mask, inp.quat[1], inp.weight[1], inp.counts, n_pat_chunk=200)
    assert np.array_equal(a["P"], b["P"])            # chunks are independent in stages 2-3 (G9)
    assert np.abs(a["model"] - b["model"]).max() <= 1e-6 * np.abs(a["model"]).max()
    assert abs(a["LL"] - b["LL"]) < 1e-9 * abs(a["LL"])


def test_masked_counts_never_matter():
    inp = make_inputs("T1")
    a = o.iterate(inp.model_init, inp.q, inp.mask, inp.quat[0], inp.weight[0], inp.counts)
    k2 = inp.counts.copy()
    k2[:, inp.mask == 0] = 7
    b = o.iterate(inp.model_init, inp.q, inp.mask, inp.quat[0], inp.weight[0], k2)
    assert np.array_equal(a["model"], b["model"]) and np.array_equal(a["P"], b["P"])


def test_normalize_underflow_conventions():
    """G20.  By default the oracle does nothing about float32 underflow: normalize returns the soft-max itself (pinned
    against the exact quotient, no value touched) and P becomes float32 by numpy's own cast at the stage boundary (gradual
    underflow).  p_min = P_MIN_FLUSH selects flush-to-zero storage, libemc's convention: what float32 holds as a normal
    number (>= 2^-126) is kept with full precision, what would be a float32 subnormal is 0, a row made only of such values
    has s = 0.  Pinned against numpy's own float32: the kept set is exactly {p : float32(p) is a normal number}."""
    assert o.P_MIN == 0.0 and o.P_MIN_FLUSH == 2.0 ** -126 == float(np.finfo(np.float32).tiny)
    # ln 2^-126 = -87.34: e^-87 is a normal float32, e^-88 and e^-100 are subnormal, e^-104 underflows float32 altogether
    big_l = np.array([[0.0, 0.0, 0.0], [-60.0, -88.0, -104.0], [-87.0, -100.0, -86.0]], np.float32)
    exact = np.exp(big_l.astype(np.float64)) / np.exp(big_l.astype(np.float64)).sum(axis=0)
    p, s, _ = o.normalize(big_l, np.full(3, 1 / 3, np.float32))
    assert np.all(p > 0) and np.allclose(p, exact, rtol=1e-14) and np.allclose(s, exact.sum(axis=1), rtol=1e-14)
    p32 = p.astype(np.float32)                                     # the stage boundary: subnormals kept, 0 below 2^-150
    assert p32[1, 1] > 0 and p32[2, 1] > 0 and p32[1, 2] == 0
    p, s, _ = o.normalize(big_l, np.full(3, 1 / 3, np.float32), p_min=o.P_MIN_FLUSH)
    normal = exact.astype(np.float32) >= np.finfo(np.float32).tiny
    assert np.array_equal(p > 0, normal)
    assert np.allclose(p[normal], exact[normal], rtol=1e-14)
    assert p[1, 1] == 0 and p[1, 2] == 0 and p[2, 1] == 0 and p[2, 0] > 0 and p[2, 2] > 0
    assert abs(p[:, 0].sum() - 1) < 1e-12 and s[1] == p[1, 0]
    # a row entirely below the threshold drops out under flush-to-zero (s = 0) and stays in under the plain cast
    big_l = np.array([[0.0, 0.0], [-95.0, -99.0]], np.float32)
    p, s, _ = o.normalize(big_l, np.full(2, 0.5, np.float32), p_min=o.P_MIN_FLUSH)
    assert s[1] == 0 and np.all(p[0] == 1.0)
    p, s, _ = o.normalize(big_l, np.full(2, 0.5, np.float32))
    assert s[1] > 0 and np.all(p.astype(np.float32)[1] > 0)
    # iterate hands p_min through: the two conventions differ exactly on rows made of float32 subnormals
    rng = np.random.default_rng(3)
    n = 8
    model = rng.random((n, n, n)).astype(np.float32) + 0.5
    q = (rng.random((30, 3)).astype(np.float32) - 0.5) * 4
    quat = rng.standard_normal((6, 4)).astype(np.float32)
    quat /= np.linalg.norm(quat, axis=1, keepdims=True)
    counts = rng.poisson(40.0, size=(5, 30)).astype(np.int32)
    a = o.iterate(model, q, None, quat, np.full(6, 1 / 6, np.float32), counts)
    b = o.iterate(model, q, None, quat, np.full(6, 1 / 6, np.float32), counts, p_min=o.P_MIN_FLUSH)
    tiny = np.finfo(np.float32).tiny
    assert np.array_equal(b["P"], np.where(a["P"] >= tiny, a["P"], 0))
    assert np.array_equal(a["L"], b["L"]) and a["LL"] == b["LL"]


# ---------------------------------------------------------------------------------------------- rotation chunks (NEXT-2)

@pytest.mark.parametrize("chunk", [1, 7, 64, 203, 500])
def test_normalize_rotation_chunks_equals_unchunked(chunk):
    """The streamed (max, sum) merge of PAPER.md:203 gives the soft-max of the whole rotation list: chunk sizes 1, ragged,
    = R and > R; also columns whose maximum moves from chunk to chunk and a weight that is exactly 0."""
    rng = np.random.default_rng(77)
    n_rot, n_pat = 203, 41
    big_l = (rng.standard_normal((n_rot, n_pat)) * 40.0 - 300.0).astype(np.float32)
    big_l[np.arange(n_pat) * 4 % n_rot, np.arange(n_pat)] += 90.0         # maxima spread over the chunks
    w = rng.random(n_rot).astype(np.float32) + 0.05
    w[5] = 0.0
    w /= w.sum()
    with np.errstate(divide="ignore"):
        p0, s0, ll0 = o.normalize(big_l, w)
        p1, s1, ll1 = o.normalize_rotation_chunks(big_l, w, chunk)
    assert np.abs(p1 - p0).max() <= 1e-13
    assert np.abs(s1 - s0).max() <= 1e-12 and abs(ll1 - ll0) <= 1e-9 * abs(ll0)
    assert np.abs(p1.sum(axis=0) - 1.0).max() <= 1e-12 and np.all(p1[5] == 0)
    from scipy.special import softmax
    with np.errstate(divide="ignore"):
        ref = softmax(big_l.astype(np.float64) + np.log(w.astype(np.float64))[:, None], axis=0)
    assert np.abs(p1 - ref).max() <= 1e-13


@pytest.mark.parametrize("chunk,weighted", [(50, False), (64, True), (203, False), (1000, True)])
def test_iterate_rotation_chunks_equals_iterate(inputs_cache, chunk, weighted):
    """Streaming the rotation list changes nothing but the summation order: model', s and LL of the chunked iteration
    equal those of `iterate` (itself pinned above) to float32 rounding."""
    inp = inputs_cache("T1")
    a = o.iterate(inp.model_init, inp.q, inp.mask, inp.quat[0], inp.weight[0], inp.counts, weighted=weighted)
    b = o.iterate_rotation_chunks(inp.model_init, inp.q, inp.mask, inp.quat[0], inp.weight[0], inp.counts, chunk,
                                  weighted=weighted)
    assert np.abs(b["s"] - a["s"]).max() <= 1e-6 * max(1.0, a["s"].max())
    assert abs(b["LL"] - a["LL"]) <= 1e-9 * abs(a["LL"])
    cov = a["den"] >= 1e-6 * a["den"].max()
    ma, mb = a["model"].reshape(-1)[cov], b["model"].reshape(-1)[cov]
    assert np.abs(mb - ma).max() <= 2e-6 * np.abs(ma).max()
    assert np.array_equal(a["den"] > 0, b["den"] > 0)


# ---------------------------------------------------------------------------------------------- photon lists (NEXT-2)

def test_photon_list_forms_equal_the_dense_definitions(inputs_cache):
    """Stages 2 and 4 summed over the photons only are the dense sums (the zero pixels of a frame contribute -W[r,p] to L,
    nothing to the update); masked counts (sentinels) never enter a list."""
    inp = inputs_cache("T1")
    w, idx = o.expand(inp.model_init, inp.q, inp.quat[0])
    lists = o.photon_lists(inp.counts, inp.mask)
    use = inp.mask.astype(bool)
    assert all(use[px].all() and (c > 0).all() for px, c in lists)
    assert sum(len(px) for px, _ in lists) == int(((inp.counts > 0) & use[None, :]).sum())
    big_l, big_a = o.loglik(w, idx, inp.counts, inp.mask)
    l_sparse = o.loglik_photon_list(w, idx, lists, inp.mask)
    assert np.abs(l_sparse - big_l).max() <= 1e-12 * big_a.max()
    p, _, _ = o.normalize(big_l.astype(np.float32), inp.weight[0])
    wn, s = o.update(p.astype(np.float32), inp.counts, inp.mask)
    wn2, s2 = o.update_photon_list(p.astype(np.float32), lists, inp.counts.shape[1])
    assert np.array_equal(s, s2)
    assert np.abs(wn2 - wn).max() <= 1e-6 * np.abs(wn).max() and np.all(wn2[:, ~use] == 0)


def test_ladder_rotations_sizes_and_weights():
    """Input generator of NEXT-1: list sizes are eq. (2.7)'s (golden ladder), quaternions are unit with w >= 0,
    the weights are positive, non-uniform and sum to 1."""
    from emc_inputs import ladder_rotations, rotation_ladder

    for d in (1, 2, 5):
        quat, w = ladder_rotations(d, 99)
        assert len(quat) == len(w) == int(rotation_ladder(d)) == 10 * (5 * d ** 3 + d)
        assert np.allclose(np.linalg.norm(quat.astype(np.float64), axis=1), 1.0, atol=1e-6) and (quat[:, 0] >= 0).all()
        assert (w > 0).all() and abs(float(w.astype(np.float64).sum()) - 1.0) <= 1e-5 and w.max() > 1.5 * w.min()
    assert int(rotation_ladder(5)) == 6300 and int(rotation_ladder(12)) == 86520

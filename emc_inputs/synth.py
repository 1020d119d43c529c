"""Seeded synthetic EMC workloads shaped like the paper's (Table 4.1) and like
BASELINE.json `configs`.  Recipe: DESIGN.md "Input recipe".

Only numpy's PCG64 generator and library routines are used here (numpy.fft for the |FFT|^2 model,
scipy Rotation + scipy.ndimage.map_coordinates(order=1) to simulate the diffraction experiment).
None of the EMC method's own arithmetic lives in this module and it imports neither the oracle nor
the CUDA package: it is the one piece both sides may share.
"""
from __future__ import annotations

import dataclasses
import os
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass

import numpy as np
from scipy.ndimage import map_coordinates
from scipy.spatial.transform import Rotation


@dataclass(frozen=True)
class EmcConfig:
    """One workload.  `n_rot` has one entry per EMC iteration (C5 grows it per stage)."""

    name: str
    n: int                      # model grid is n^3 (64^3 / 128^3, G = P^(3/2))
    n_det: int                  # detector is n_det x n_det pixels (binned 64^2 / 128^2)
    n_rot: tuple                # rotations per iteration (PAPER.md:93-98 ladder sizes in the paper)
    n_pat: int                  # number of patterns M_data
    n_pat_chunk: int            # patterns per streamed chunk (config 4), == n_pat otherwise
    count_dtype: str            # "int32" | "uint16" | "uint8"
    mean_photons: float         # mean photons per unmasked pixel
    n_spheres: int              # Gaussian blobs in the real-space object
    beamstop_radius: float      # centred beamstop radius in pixels, 0 = none
    gap_rows: int               # horizontal panel gap height in pixels, 0 = none
    seed: int                   # config number c: seeds are 1000+c, 2000+c(+stage), 3000+c, 4000+c

    @property
    def n_iter(self) -> int:
        return len(self.n_rot)

    @property
    def n_pix(self) -> int:
        return self.n_det * self.n_det


CONFIGS = {
    # BASELINE.json configs[0..4]
    "C1": EmcConfig("C1", 32, 32, (480,), 1000, 1000, "int32", 1.0, 40, 0.0, 0, 1),
    "C2": EmcConfig("C2", 64, 64, (5000,) * 3, 10000, 10000, "uint16", 0.1, 80, 6.0, 0, 2),
    "C3": EmcConfig("C3", 128, 128, (25000,), 50000, 50000, "uint16", 0.05, 80, 6.0, 4, 3),
    "C4": EmcConfig("C4", 128, 128, (10000,), 200000, 25000, "uint16", 0.01, 80, 6.0, 4, 4),
    "C5": EmcConfig("C5", 256, 256, (2000, 5000, 10000, 25000, 50000), 20000, 20000, "uint16", 0.2,
                    80, 6.0, 0, 5),
    # small cases for CPU tests and parity runs that the oracle finishes in seconds; they keep the
    # structure (mask, ragged sizes that are no multiple of any tile) but not the size.
    "T0": EmcConfig("T0", 16, 16, (60,), 40, 40, "int32", 2.0, 12, 0.0, 0, 10),
    "T1": EmcConfig("T1", 24, 20, (203,), 157, 157, "uint16", 0.5, 20, 2.0, 2, 11),
    "T2": EmcConfig("T2", 32, 40, (333, 401), 517, 200, "uint16", 0.3, 30, 3.0, 2, 12),
    # odd everything: grid 17^3 (no blocked layouts), 15 x 15 = 225 pixels (rows of W' not 16-byte aligned), uint8 counts
    "T3": EmcConfig("T3", 17, 15, (97,), 77, 77, "uint8", 0.8, 10, 1.5, 1, 13),
}


@dataclass
class EmcInputs:
    cfg: EmcConfig
    model_true: np.ndarray      # [n,n,n] float32, z fastest, DC bin at (n/2,n/2,n/2)
    model_init: np.ndarray      # [n,n,n] float32 = model_true * seeded log-normal noise
    q: np.ndarray               # [P,3] float32, Ewald-sphere pixel coordinates in voxel units
    mask: np.ndarray            # [P] uint8, 1 = use
    quat: list                  # per stage: [R,4] float32 (w,x,y,z), unit, w >= 0
    weight: list                # per stage: [R] float32, sums to 1
    counts: np.ndarray          # [N,P] photon counts (masked pixels hold a sentinel)
    r_true: np.ndarray          # [N] index into quat[-1] of the generating rotation


def rotation_ladder(d):
    """Eq (2.7): M_rot(d) = 10 (5 d^3 + d)."""
    d = np.asarray(d, dtype=np.int64)
    return 10 * (5 * d ** 3 + d)


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def blob_object(n: int, n_spheres: int, seed: int) -> np.ndarray:
    """Real-space density: Gaussian blobs with centres uniform in a ball of radius n/4 around the
    grid centre, sigma ~ U[0.8, 1.6] voxels, amplitude ~ U[0.5, 1]."""
    rng = _rng(seed)
    # uniform in a ball: direction from normals, radius ~ U^(1/3)
    v = rng.standard_normal((n_spheres, 3))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    rad = (n / 4.0) * rng.random(n_spheres) ** (1.0 / 3.0)
    centre = n / 2.0 + v * rad[:, None]
    sigma = rng.uniform(0.8, 1.6, n_spheres)
    amp = rng.uniform(0.5, 1.0, n_spheres)
    ax = np.arange(n, dtype=np.float64)
    rho = np.zeros((n, n, n), dtype=np.float64)
    for c, s, a in zip(centre, sigma, amp):
        gx = np.exp(-0.5 * ((ax - c[0]) / s) ** 2)
        gy = np.exp(-0.5 * ((ax - c[1]) / s) ** 2)
        gz = np.exp(-0.5 * ((ax - c[2]) / s) ** 2)
        rho += a * gx[:, None, None] * gy[None, :, None] * gz[None, None, :]
    return rho


def intensity_model(rho: np.ndarray) -> np.ndarray:
    """|FFT|^2 of the object, fft-shifted so the DC bin sits at index n/2 on every axis."""
    f = np.fft.fftn(np.fft.ifftshift(rho))
    return np.fft.fftshift(np.abs(f) ** 2)


def detector_geometry(n_det: int, n: int) -> np.ndarray:
    """Ewald-sphere pixel coordinates q [P,3] in voxel units.

    Flat detector at distance D = n_det pixels; pixel centres x,y = index - (n_det-1)/2;
    q~ = (x/rho, y/rho, D/rho - 1) with rho = sqrt(x^2+y^2+D^2); scaled so that the largest |q|
    (corner pixel) is n/2 - 1 voxels."""
    ax = np.arange(n_det, dtype=np.float64) - (n_det - 1) / 2.0
    y, x = np.meshgrid(ax, ax, indexing="ij")       # row index = y, column index = x; p = row*n_det+col
    dist = float(n_det)
    rho = np.sqrt(x * x + y * y + dist * dist)
    qt = np.stack([x / rho, y / rho, dist / rho - 1.0], axis=-1).reshape(-1, 3)
    scale = (n / 2.0 - 1.0) / np.sqrt((qt * qt).sum(axis=1)).max()
    return (qt * scale).astype(np.float32)


def detector_mask(n_det: int, beamstop_radius: float, gap_rows: int) -> np.ndarray:
    """1 = use.  Beamstop: pixels with x^2+y^2 <= r^2; panel gap: the `gap_rows` central rows."""
    ax = np.arange(n_det, dtype=np.float64) - (n_det - 1) / 2.0
    y, x = np.meshgrid(ax, ax, indexing="ij")
    mask = np.ones((n_det, n_det), dtype=np.uint8)
    if beamstop_radius > 0:
        mask[x * x + y * y <= beamstop_radius * beamstop_radius] = 0
    if gap_rows > 0:
        lo = n_det // 2 - gap_rows // 2
        mask[lo:lo + gap_rows, :] = 0
    return mask.reshape(-1)


def random_rotations(n_rot: int, seed: int) -> np.ndarray:
    """Uniform random unit quaternions (w,x,y,z): 4 standard normals, normalised, w >= 0."""
    rng = _rng(seed)
    v = rng.standard_normal((n_rot, 4))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    v[v[:, 0] < 0] *= -1.0
    return v.astype(np.float32)


def ladder_rotations(d: int, seed: int):
    """A rotation list of the size eq. (2.7) gives for discretisation level d, M_rot(d) = 10 (5 d^3 + d) (PAPER.md:95-98:
    6 300 for d = 5 ... 86 520 for d = 12), WITH non-uniform prior weights w_j.  The paper refines the
    600-cell (ref. [11] App. C, not in the container); the stand-in is seeded uniform random quaternions, each weighted by
    the volume it represents: w_j ~ (distance to its nearest neighbour on the 3-sphere, antipodes identified)^3,
    normalised to sum 1 (a library nearest-neighbour query, scipy cKDTree).  Returns (quat [M,4] float32, weight [M] float32)."""
    from scipy.spatial import cKDTree

    m = int(rotation_ladder(d))
    quat = random_rotations(m, seed)
    both = np.concatenate([quat, -quat]).astype(np.float64)       # q and -q are the same rotation
    dist, _ = cKDTree(both).query(quat.astype(np.float64), k=2)
    w = dist[:, 1] ** 3
    return quat, (w / w.sum()).astype(np.float32)


def _slices_library(model64: np.ndarray, q: np.ndarray, quat: np.ndarray) -> np.ndarray:
    """Mean intensities of the simulated experiment: the model read at R q + n/2 by the library's
    own linear interpolation.  scipy's quaternions are scalar-last."""
    n = model64.shape[0]
    rot = Rotation.from_quat(np.asarray(quat, dtype=np.float64)[:, [1, 2, 3, 0]])
    mats = rot.as_matrix()                                    # [D,3,3]
    x = np.einsum("dab,pb->adp", mats, q.astype(np.float64)) + n / 2.0   # [3,D,P]
    lam = map_coordinates(model64, x.reshape(3, -1), order=1, mode="constant", cval=0.0)
    return lam.reshape(len(quat), len(q))


_SENTINEL = {"int32": 2 ** 31 - 1, "uint16": 65535, "uint8": 255}


_CHUNK = 256        # patterns per Poisson stream: part of the recipe (the counts do not depend on the thread count)


def simulate_patterns(model64, q, mask, quat_list, n_pat, mean_photons, count_dtype, seed_orient,
                      seed_poisson):
    """Poisson photon counts of n_pat shots at orientations drawn uniformly from `quat_list`.
    Chunk c of 256 consecutive patterns draws from its own PCG64 stream seeded (seed_poisson, c), so the
    chunks can be generated by several threads (the scipy / numpy routines release the GIL) with the
    same result on any machine.

    Returns (counts [N,P], r_true [N], scale): `scale` is the factor by which the model has to be
    multiplied so that the mean expected count over unmasked pixels is `mean_photons`."""
    r_true = _rng(seed_orient).integers(0, len(quat_list), n_pat)
    use = mask.astype(bool)
    # pass 1: scale from a bounded sample of the shots (exact mean for small N)
    probe = r_true[: min(n_pat, 512)]
    lam = _slices_library(model64, q, quat_list[probe])
    scale = mean_photons / lam[:, use].mean()
    counts = np.empty((n_pat, len(q)), dtype=count_dtype)
    hi = np.iinfo(count_dtype).max
    sentinel = _SENTINEL[count_dtype]

    def one_chunk(c):
        d0 = c * _CHUNK
        d1 = min(n_pat, d0 + _CHUNK)
        rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence((seed_poisson, c))))
        lam = _slices_library(model64, q, quat_list[r_true[d0:d1]]) * scale
        k = rng.poisson(np.maximum(lam, 0.0))
        block = np.minimum(k, hi - 1).astype(count_dtype)
        block[:, ~use] = sentinel                   # garbage that every stage must ignore (G16)
        counts[d0:d1] = block

    n_chunks = -(-n_pat // _CHUNK)
    workers = max(1, min(32, os.cpu_count() or 1, n_chunks))
    if workers == 1:
        for c in range(n_chunks):
            one_chunk(c)
    else:
        with ThreadPoolExecutor(workers) as pool:
            list(pool.map(one_chunk, range(n_chunks)))
    return counts, r_true.astype(np.int32), float(scale)


def make_inputs(cfg: EmcConfig | str, n_pat: int | None = None) -> EmcInputs:
    """Build the whole seeded workload of a config.  `n_pat` overrides the pattern count (bounded
    samples of a big config keep every other shape)."""
    if isinstance(cfg, str):
        cfg = CONFIGS[cfg]
    if n_pat is not None:
        cfg = dataclasses.replace(cfg, n_pat=n_pat, n_pat_chunk=min(cfg.n_pat_chunk, n_pat))
    c = cfg.seed
    rho = blob_object(cfg.n, cfg.n_spheres, 1000 + c)
    model64 = intensity_model(rho)
    q = detector_geometry(cfg.n_det, cfg.n)
    mask = detector_mask(cfg.n_det, cfg.beamstop_radius, cfg.gap_rows)
    quat = []
    for s, r in enumerate(cfg.n_rot):       # a fresh list only when the stage changes R (C5)
        same = s > 0 and r == cfg.n_rot[s - 1]
        quat.append(quat[-1] if same else random_rotations(r, 2000 + c + 100 * s))
    weight = [np.full(r, 1.0 / r, dtype=np.float32) for r in cfg.n_rot]
    counts, r_true, scale = simulate_patterns(model64, q, mask, quat[-1], cfg.n_pat, cfg.mean_photons,
                                              cfg.count_dtype, 3000 + c, 4000 + c)
    model_true = (model64 * scale).astype(np.float32)
    noise = np.exp(0.5 * _rng(5000 + c).standard_normal(model_true.shape))
    model_init = (model64 * scale * noise).astype(np.float32)
    return EmcInputs(cfg, model_true, model_init, q, mask, quat, weight, counts, r_true)

"""End-to-end gates on model' for the GPU parity tests, aware of reading G20.

The oracle leaves the float32 responsibilities to the plain cast (gradual underflow, oracle.P_MIN = 0); libemc stores them
flush-to-zero below 2^-126 (EMC_P_MIN).  The two differ only on FRAGILE slices: rotations whose weights s[r] = sum_d P[r,d]
hang on float32 subnormals.  Such a slice has no responsibility with 24 significant bits left, so its W' cannot be formed
to T3's 1e-5 by any float32 pipeline; under eq. (2.12) it weighs < 2^-126 N and does not matter, under eq. (2.10) it has
weight 1 on the voxels it touches.  The gates therefore
  * require the SAME set of slices with s[r] > 0 on both sides, except fragile ones,
  * hold every voxel that no fragile slice touches to a tight bound,
  * bound the voxels a fragile slice does touch by that slice's share of the voxel's summed weights.
Nothing here is shared with the CUDA path; the oracle is called for the fragile slices' footprint only.
"""
import numpy as np

from oracle import emc_oracle as o

TINY = float(np.finfo(np.float32).tiny)      # 2^-126


def flushed(p32):
    """P as libemc stores it: float32 subnormals are 0 (EMC_P_MIN, include/emc.h)."""
    p32 = np.asarray(p32, dtype=np.float32)
    return np.where(p32 >= TINY, p32, np.float32(0))


def fragile_rows(p32, dl_max=0.0):
    """Rows of the oracle's float32 P whose s[r] depends on float32's underflow convention by more than 1e-6 relative, or
    whose largest responsibility lies within the measured log-likelihood difference of the flush threshold (P on the two
    sides differ by at most a factor exp(2 dl_max), DESIGN.md section 4 T2): the slices whose status may legitimately
    differ between the plain float32 cast and flush-to-zero storage."""
    p32 = np.asarray(p32, dtype=np.float32)
    pd = p32.astype(np.float64)
    s = pd.sum(axis=1)
    sub = np.where(p32 < TINY, pd, 0.0).sum(axis=1)
    edge = p32.max(axis=1) < TINY * np.exp(2.0 * dl_max)
    return (s > 0) & ((sub > 1e-6 * s) | edge)


def footprint(rows, q, quat, mask, n):
    """den of eq. (2.10) restricted to the given rotations: > 0 exactly on the voxels they touch."""
    if not np.any(rows):
        return np.zeros(n ** 3)
    k = int(np.count_nonzero(rows))
    _, _, den = o.compress(np.ones((k, np.asarray(q).shape[0]), np.float32), q, np.asarray(quat)[rows], mask, n)
    return den


def edge_rows(p32_cast, dl_max):
    """Rows of the plain-cast oracle's P whose largest responsibility lies within a factor exp(2 dl_max) of 2^-126 on either
    side: the slices whose flush-to-zero status may differ between two evaluations whose L differ by dl_max."""
    mx = np.asarray(p32_cast, dtype=np.float32).max(axis=1).astype(np.float64)
    return (mx >= TINY * np.exp(-2.0 * dl_max)) & (mx < TINY * np.exp(2.0 * dl_max))


def model_gate(m, ref, weighted, q, quat, mask, count_max, s_gpu=None, dl_max=0.0, tight=2e-3, label="", fragile=None):
    """m: the GPU's model'; ref: oracle.iterate(...) at its default (plain float32 cast of P).  `fragile` overrides the
    classification (for a `ref` computed with p_min = P_MIN_FLUSH: pass edge_rows of the plain-cast P).
    Measured on a B200 (round 3): worst clean voxel 1.2e-3 (C1), 2.0e-4 (T2), 1.6e-4 (C2); hence tight = 2e-3."""
    n = ref["model"].shape[0]
    m, m_ref = np.asarray(m).reshape(-1).astype(np.float64), ref["model"].reshape(-1).astype(np.float64)
    den = ref["den"]
    frag = fragile_rows(ref["P"], dl_max) if fragile is None else np.asarray(fragile, dtype=bool)
    if s_gpu is not None:
        differ = (np.asarray(s_gpu) > 0) != (ref["s"] > 0)
        assert not np.any(differ & ~frag), f"{int((differ & ~frag).sum())} slices change status away from float32's underflow edge"
    cov = den >= 1e-3 * den.max()
    scale = np.abs(m_ref).max()
    rel = np.abs(m - m_ref) / (np.abs(m_ref) + 1e-6 * scale)
    den_f = footprint(frag, q, quat, mask, n) if not weighted else np.zeros_like(den)
    clean = cov & (den_f == 0)
    worst = rel[clean].max(initial=0.0)
    med = float(np.median(rel[clean])) if clean.any() else 0.0
    print(f"model gate {label}: fragile slices {int(frag.sum())}, voxels they touch {int((cov & ~clean).sum())} of {int(cov.sum())}; "
          f"rel error elsewhere max {worst:.2e}, median {med:.2e} (median over all covered voxels {np.median(rel[cov]):.2e})")
    assert worst <= tight, f"max rel model error {worst:.3e} on voxels no fragile slice touches"
    assert med <= 1e-4, f"median rel model error {med:.3e} on voxels no fragile slice touches"
    # a fragile slice enters den[l] with at most den_f[l] and num[l] with at most den_f[l] * (largest count): whether and
    # how it takes part moves model'[l] by no more than its share of the voxel's weights times that range
    touched = cov & ~clean
    if touched.any():
        share = den_f[touched] / np.maximum(den[touched] - den_f[touched], 1e-30)
        bound = 2.0 * share * (count_max + np.abs(m_ref[touched])) + tight * (np.abs(m_ref[touched]) + 1e-6 * scale)
        assert np.all(np.abs(m - m_ref)[touched] <= bound), "a voxel moved by more than the fragile slices' share of it"
    assert np.all(m[den == 0] == 0)

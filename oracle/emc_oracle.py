"""CPU ORACLE for one EMC iteration (Expand -> Poisson log-likelihood -> normalise -> update ->
Compress).  TEST INFRASTRUCTURE ONLY.

This file is the plain, slow, obviously-correct restatement of what the CUDA path in
`paper_1409_4256_b200/` must compute.  It is written from the paper and the readings in
DESIGN.md §3, shares no code with the CUDA path, and may be imported only by `tests/`,
`__graft_entry__.smoke()`, `bench.py`'s `cpu_baseline` leg and `bench.py --impl reference`.

Every stage is a *direct formula*, so each function is that definition written out with numpy:
fp32 inputs and outputs (the paper works in single precision), float64 arithmetic
and accumulation inside.  Library primitives used as steps: numpy's float64 matmul, np.bincount
(weighted scatter-add), np.exp/np.log.  No blocking, fusion or reordering beyond the formulas.

Pins (tests/test_oracle_*.py, `-m "not gpu"`): every function below is pinned by closed forms,
brute force on tiny inputs, invariants and independent library routines (scipy Rotation,
scipy.ndimage.map_coordinates, scipy.stats.poisson, scipy.special.softmax/logsumexp); the table is
in DESIGN.md §5.  The paper prints no worked numeric example of any stage, so no pin is a printed
value (tests/golden/ holds only eq. (2.7)'s printed ladder).  No function is "parity unpinned".

Notation (paper -> here): M_rot -> R (index r), M_data -> N (index d), M_pix -> P (index p),
M_grid -> G = n^3 (index l); W_ij -> W[r,p]; blackboard W_l -> model[l]; P_jk -> P[r,d]; w_j -> w[r].
"""
from __future__ import annotations

import numpy as np

LOGW_FLOOR = np.float32(1e-30)      # DESIGN.md §3 G8: log(max(W, 1e-30))
# DESIGN.md §3 G20.  P is a float32 quantity and the paper says nothing about its underflow, so
# the oracle does nothing about it either: P_MIN = 0 leaves P to the plain float32 cast at the stage boundary (IEEE
# gradual underflow: subnormals kept, 0 below 2^-150).  P_MIN_FLUSH = 2^-126 names the other float32 convention,
# flush-to-zero below the smallest normal number, which is what libemc's storage does (EMC_P_MIN in include/emc.h);
# tests select it with the `p_min` argument where they examine that convention.  The default is the plain cast.
P_MIN = 0.0
P_MIN_FLUSH = float(np.finfo(np.float32).tiny)


# ----------------------------------------------------------------------------------------------
# Geometry: rotation, sample coordinates, base-corner index map   (eq. 2.9's argument R_j q_i)
# ----------------------------------------------------------------------------------------------

def rotation_matrix(quat):
    """Active rotation matrix of a unit quaternion (w,x,y,z); PAPER.md:93 ("quaternions encode
    rotations"), PAPER.md:66 (the sample position is R_j q_i).

    Textbook formula, evaluated in float64 from the float32 components, every entry rounded once
    to float32 (DESIGN.md §3 G4).  Returns [R,3,3] float32."""
    qd = np.asarray(quat, dtype=np.float32).astype(np.float64)
    w, x, y, z = qd[..., 0], qd[..., 1], qd[..., 2], qd[..., 3]
    m = np.empty(qd.shape[:-1] + (3, 3), dtype=np.float64)
    m[..., 0, 0] = 1.0 - 2.0 * (y * y + z * z)
    m[..., 0, 1] = 2.0 * (x * y - w * z)
    m[..., 0, 2] = 2.0 * (x * z + w * y)
    m[..., 1, 0] = 2.0 * (x * y + w * z)
    m[..., 1, 1] = 1.0 - 2.0 * (x * x + z * z)
    m[..., 1, 2] = 2.0 * (y * z - w * x)
    m[..., 2, 0] = 2.0 * (x * z - w * y)
    m[..., 2, 1] = 2.0 * (y * z + w * x)
    m[..., 2, 2] = 1.0 - 2.0 * (x * x + y * y)
    return m.astype(np.float32)


def sample_coords(quat, q, n):
    """Grid coordinates x[r,p,:] = R_r q_p + c of every sample, c = n/2 (DESIGN.md §3 G5).

    float32 arithmetic with every multiply and add rounded separately, in this order
    (DESIGN.md §3 G4 -- this sequence is what makes the index map bit-exact on any machine):
        x_a = ((R_a0*q_x + R_a1*q_y) + R_a2*q_z) + c
    Returns [R,P,3] float32."""
    rm = rotation_matrix(quat)                                  # [R,3,3] f32
    q = np.asarray(q, dtype=np.float32)
    c = np.float32(n / 2.0)
    qx, qy, qz = q[None, :, 0], q[None, :, 1], q[None, :, 2]
    out = np.empty((rm.shape[0], q.shape[0], 3), dtype=np.float32)
    for a in range(3):
        t0 = rm[:, a, 0, None] * qx                             # each op is one float32 rounding
        t1 = rm[:, a, 1, None] * qy
        t2 = rm[:, a, 2, None] * qz
        out[:, :, a] = ((t0 + t1) + t2) + c
    return out


def base_corner(x, n):
    """Base corner b = floor(x), fractional offsets t = x - b, validity and linear index.

    Valid iff 0 <= b_a <= n-2 on all three axes (all 8 neighbours exist; DESIGN.md §3 G7).
    idx = (b_x*n + b_y)*n + b_z (z fastest, G5) or -1.  Returns (b int32, t float32, valid, idx)."""
    b = np.floor(x)
    t = (x - b).astype(np.float32)                              # exact in float32
    b = b.astype(np.int32)
    valid = np.all((b >= 0) & (b <= n - 2), axis=-1)
    idx = (b[..., 0].astype(np.int64) * n + b[..., 1]) * n + b[..., 2]
    idx = np.where(valid, idx, -1).astype(np.int32)
    return b, t, valid, idx


def index_map(quat, q, n):
    """The rotation -> voxel index map idx[r,p] (int32, -1 outside the grid).  Bit-exact target."""
    return base_corner(sample_coords(quat, q, n), n)[3]


def _corner_weights(t):
    """Trilinear weights f for the 8 corners (i,j,k) in {0,1}^3, as float64 [..., 8] in the order
    corner = 4i + 2j + k; per axis the weight is (1 - t) for offset 0 and t for offset 1.
    This is the interpolation kernel f of eq. (2.8), PAPER.md:106-109 (f := trilinear, G-A9)."""
    td = t.astype(np.float64)
    w0 = 1.0 - td
    w1 = td
    ws = []
    for i in (0, 1):
        for j in (0, 1):
            for k in (0, 1):
                ws.append((w1 if i else w0)[..., 0] * (w1 if j else w0)[..., 1] * (w1 if k else w0)[..., 2])
    return np.stack(ws, axis=-1)


def _corner_offsets(n):
    return np.array([(i * n + j) * n + k for i in (0, 1) for j in (0, 1) for k in (0, 1)], dtype=np.int64)


# ----------------------------------------------------------------------------------------------
# Stage 1: Expand (e-step), eq. (2.9)
# ----------------------------------------------------------------------------------------------

def expand(model, q, quat, chunk=64):
    """W[r,p] = sum_l f(p_l - R_r q_p) model[l]  (eq. 2.9): trilinear read of the model at every
    sample; samples outside the grid give W = 0 (G7).  Computed for every pixel, masked or not.
    Returns (W [R,P] float32, idx [R,P] int32)."""
    model = np.asarray(model, dtype=np.float32)
    n = model.shape[0]
    flat = model.reshape(-1).astype(np.float64)
    quat = np.asarray(quat, dtype=np.float32)
    n_rot, n_pix = quat.shape[0], np.asarray(q).shape[0]
    w_out = np.zeros((n_rot, n_pix), dtype=np.float32)
    idx_out = np.empty((n_rot, n_pix), dtype=np.int32)
    off = _corner_offsets(n)
    for r0 in range(0, n_rot, chunk):
        r1 = min(n_rot, r0 + chunk)
        _, t, valid, idx = base_corner(sample_coords(quat[r0:r1], q, n), n)
        f = _corner_weights(t)                                  # [r,P,8]
        base = np.where(valid, idx, 0).astype(np.int64)
        vals = flat[base[..., None] + off]                      # [r,P,8]
        w = (f * vals).sum(axis=-1)
        w_out[r0:r1] = np.where(valid, w, 0.0).astype(np.float32)
        idx_out[r0:r1] = idx
    return w_out, idx_out


# ----------------------------------------------------------------------------------------------
# Stage 2: Poisson log-likelihood, north_star formula; Poisson model of PAPER.md:68
# ----------------------------------------------------------------------------------------------

def log_slices(w, idx):
    """logW[r,p] = log(max(W, 1e-30)) for samples inside the grid, 0 outside (G7, G8)."""
    w = np.asarray(w, dtype=np.float32)
    lw = np.log(np.maximum(w, LOGW_FLOOR).astype(np.float64))
    return np.where(np.asarray(idx) >= 0, lw, 0.0)


def loglik(w, idx, counts, mask):
    """L[r,d] = sum_p mask_p (K[d,p] log W[r,p] - W[r,p])   (north_star stage 2; the -log K! term of
    the Poisson pmf is constant in r and dropped, G2).

    Also returns A[r,d] = sum_p mask_p (K |log W| + W), the scale the L tolerance refers to
    (DESIGN.md §4 T1).  Returns (L float64 [R,N], A float64 [R,N])."""
    use = _use(mask, np.asarray(w).shape[1])
    wd = np.asarray(w, dtype=np.float32).astype(np.float64)[:, use]
    lw = log_slices(w, idx)[:, use]
    k = np.asarray(counts)[:, use].astype(np.float64)           # [N,Pu]
    s = wd.sum(axis=1)
    big_l = lw @ k.T - s[:, None]
    big_a = np.abs(lw) @ k.T + np.abs(wd).sum(axis=1)[:, None]
    return big_l, big_a


def _use(mask, n_pix):
    if mask is None:
        return np.ones(n_pix, dtype=bool)
    return np.asarray(mask).astype(bool)


# ----------------------------------------------------------------------------------------------
# Stage 3: normalisation over rotations (reconstructed eq. 2.4)
# ----------------------------------------------------------------------------------------------

def normalize(big_l, weight, p_min=None):
    """P[r,d] = w_r T_rd / sum_r' w_r' T_r'd with T = exp(L), evaluated max-subtracted
    ("some care ... finite precision"; only max and sum are needed):
        a = L + log w_r;  m_d = max_r a;  e = exp(a - m_d);  P = e / sum_r e.
    Values below `p_min` (default P_MIN = 0: none) are returned as 0: p_min = P_MIN_FLUSH = 2^-126 is the
    flush-to-zero storage of float32 (G20); a rotation whose whole row is 0 has s[r] = 0 and is skipped
    by Compress (G17).
    Also s[r] = sum_d P[r,d] and the total log-likelihood LL = sum_d (m_d + log sum_r e).
    `big_l` is taken as given (tests feed the float32-rounded L, DESIGN.md §4 T2).
    Returns (P float64 [R,N], s float64 [R], LL float)."""
    a = np.asarray(big_l).astype(np.float64) + np.log(np.asarray(weight).astype(np.float64))[:, None]
    m = a.max(axis=0)
    e = np.exp(a - m[None, :])
    z = e.sum(axis=0)
    p = e / z[None, :]
    p[p < (P_MIN if p_min is None else p_min)] = 0.0            # G20 (a no-op at the default)
    return p, p.sum(axis=1), float((m + np.log(z)).sum())


# ----------------------------------------------------------------------------------------------
# Stage 4: slice update (M-step), eq. (2.5) with phi == 1 / eq. (2.11)
# ----------------------------------------------------------------------------------------------

def update(p, counts, mask):
    """W'[r,p] = sum_d P[r,d] K[d,p] / sum_d P[r,d]   (eq. 2.5 with the printed index typo read as
    P_jk, G10).  Masked pixels give 0 (G16); rows with s[r] = 0 give 0 (G17).
    `p` is taken as given (the float32 responsibilities).  Returns (W' float32 [R,P], s float64)."""
    pd = np.asarray(p).astype(np.float64)
    k = np.asarray(counts)
    use = _use(mask, k.shape[1])
    s = pd.sum(axis=1)
    num = pd @ np.where(use[None, :], k, 0).astype(np.float64)  # eq. (2.11)
    with np.errstate(divide="ignore", invalid="ignore"):
        wn = np.where(s[:, None] > 0, num / s[:, None], 0.0)
    wn[:, ~use] = 0.0
    return wn.astype(np.float32), s


# ----------------------------------------------------------------------------------------------
# Stage 5: Compress (c-step), eq. (2.10) / (2.12)
# ----------------------------------------------------------------------------------------------

def compress(wn, q, quat, mask, n, slice_w=None, chunk=64):
    """model'[l] = sum_{r,p} f(p_l - R_r q_p) om_r W'[r,p] / sum_{r,p} f(p_l - R_r q_p) om_r
    over unmasked samples inside the grid, 0 where the denominator is 0 (G17).

    om_r = 1 (and slices with slice_w[r] == 0 skipped) is eq. (2.10); om_r = s[r] = sum_d P[r,d]
    applied to numerator and denominator is exactly eq. (2.12) with W' normalised (G6).  The
    numerator and denominator are accumulated separately, the division is last.
    `slice_w` None = all ones.  `weighted` selection is the caller's: pass om_r itself.
    Returns (model' float32 [n,n,n], num float64 [G], den float64 [G])."""
    wn = np.asarray(wn, dtype=np.float32)
    quat = np.asarray(quat, dtype=np.float32)
    n_rot, n_pix = wn.shape
    use = _use(mask, n_pix)
    om = np.ones(n_rot, dtype=np.float64) if slice_w is None else np.asarray(slice_w).astype(np.float64)
    g = n * n * n
    num = np.zeros(g, dtype=np.float64)
    den = np.zeros(g, dtype=np.float64)
    off = _corner_offsets(n)
    for r0 in range(0, n_rot, chunk):
        r1 = min(n_rot, r0 + chunk)
        _, t, valid, idx = base_corner(sample_coords(quat[r0:r1], q, n), n)
        take = valid & use[None, :] & (om[r0:r1, None] > 0)
        f = _corner_weights(t)[take] * np.broadcast_to(om[r0:r1, None], valid.shape)[take][:, None]
        tgt = idx[take].astype(np.int64)[:, None] + off[None, :]
        val = wn[r0:r1].astype(np.float64)[take]
        num += np.bincount(tgt.reshape(-1), weights=(f * val[:, None]).reshape(-1), minlength=g)
        den += np.bincount(tgt.reshape(-1), weights=f.reshape(-1), minlength=g)
    with np.errstate(divide="ignore", invalid="ignore"):
        model = np.where(den > 0, num / den, 0.0)
    return model.astype(np.float32).reshape(n, n, n), num, den


# ----------------------------------------------------------------------------------------------
# One iteration (Algorithm 1), with pattern chunks (config 4, G9)
# ----------------------------------------------------------------------------------------------

def iterate(model, q, mask, quat, weight, counts, n_pat_chunk=None, weighted=False, p_min=None):
    """expand -> [per pattern chunk: loglik -> normalize] -> update -> compress.

    Stage boundaries carry float32 (W, L, P, W'), as the C-ABI does.  The soft-max is over
    rotations per pattern, so pattern chunks are independent in stages 2-3; s[r] and the update
    numerators add up over chunks and are divided after the last one (G9).
    `weighted` selects eq. (2.12) (om_r = s[r]) instead of eq. (2.10) (om_r = 1).
    `p_min`: see normalize (default: the plain float32 cast of P).
    Returns dict(model, W, idx, L, P, s, Wn, LL)."""
    counts = np.asarray(counts)
    n = np.asarray(model).shape[0]
    n_pat = counts.shape[0]
    chunk = n_pat if not n_pat_chunk else n_pat_chunk
    w, idx = expand(model, q, quat)
    use = _use(mask, counts.shape[1])
    l_all = np.empty((w.shape[0], n_pat), dtype=np.float32)
    p_all = np.empty((w.shape[0], n_pat), dtype=np.float32)
    s = np.zeros(w.shape[0], dtype=np.float64)
    num = np.zeros(w.shape, dtype=np.float64)
    ll = 0.0
    for d0 in range(0, n_pat, chunk):
        d1 = min(n_pat, d0 + chunk)
        big_l, _ = loglik(w, idx, counts[d0:d1], mask)
        l32 = big_l.astype(np.float32)
        p, _, ll_c = normalize(l32, weight, p_min)
        p32 = p.astype(np.float32)
        l_all[:, d0:d1] = l32
        p_all[:, d0:d1] = p32
        ll += ll_c
        pd = p32.astype(np.float64)
        s += pd.sum(axis=1)
        num += pd @ np.where(use[None, :], counts[d0:d1], 0).astype(np.float64)
    with np.errstate(divide="ignore", invalid="ignore"):
        wn = np.where(s[:, None] > 0, num / s[:, None], 0.0)
    wn[:, ~use] = 0.0
    wn = wn.astype(np.float32)
    om = s.astype(np.float32) if weighted else (s > 0).astype(np.float32)
    new_model, _, den = compress(wn, q, quat, mask, n, slice_w=om)
    return dict(model=new_model, W=w, idx=idx, L=l_all, P=p_all, s=s, Wn=wn, LL=ll, den=den)


# ----------------------------------------------------------------------------------------------
# Photon-list form of stages 2 and 4 for sparse frames (BASELINE.json config 4: > 99 % of the pixels hold no
# photon; DESIGN.md section 11 NEXT-2).  Same sums as `loglik` / `update`, taken over the photons only.
# ----------------------------------------------------------------------------------------------

def photon_lists(counts, mask):
    """Per pattern d the list of (pixel p, count K[d,p]) over unmasked pixels with K[d,p] > 0."""
    counts = np.asarray(counts)
    use = _use(mask, counts.shape[1])
    out = []
    for row in counts:
        px = np.nonzero((row > 0) & use)[0]
        out.append((px, row[px].astype(np.float64)))
    return out


def loglik_photon_list(w, idx, lists, mask):
    """L[r,d] = sum_{(p,c) in list d} c logW[r,p] - sum_{p: mask} W[r,p]   (the zero pixels of a frame only
    contribute -W[r,p], which is the same for every frame).  Returns L float64 [R,N]."""
    use = _use(mask, np.asarray(w).shape[1])
    lw = log_slices(w, idx)
    s = np.asarray(w, dtype=np.float32).astype(np.float64)[:, use].sum(axis=1)
    big_l = np.empty((lw.shape[0], len(lists)))
    for d, (px, c) in enumerate(lists):
        big_l[:, d] = lw[:, px] @ c - s
    return big_l


def update_photon_list(p, lists, n_pix):
    """W'[r,p] = sum_d P[r,d] K[d,p] / sum_d P[r,d], the numerator scattered photon by photon (eq. 2.11)."""
    pd = np.asarray(p).astype(np.float64)
    num = np.zeros((pd.shape[0], n_pix))
    for d, (px, c) in enumerate(lists):
        num[:, px] += pd[:, d:d + 1] * c[None, :]
    s = pd.sum(axis=1)
    with np.errstate(divide="ignore", invalid="ignore"):
        wn = np.where(s[:, None] > 0, num / s[:, None], 0.0)
    return wn.astype(np.float32), s


# ----------------------------------------------------------------------------------------------
# Rotation chunks (the paper's own streaming, "chunk C_c", 203; DESIGN.md section 11 NEXT-2)
# ----------------------------------------------------------------------------------------------

def _merge_max_sum(m, z, a):
    """(m, z) <- merged with the (max, sum) of the rows `a` of one chunk.  A column in which nothing
    finite has been seen yet (zero weights: a = -inf) carries m = -inf, z = 0."""
    m_c = a.max(axis=0)
    live_c, live = np.isfinite(m_c), np.isfinite(m)
    with np.errstate(invalid="ignore"):
        z_c = np.where(live_c, np.exp(a - np.where(live_c, m_c, 0.0)[None, :]).sum(axis=0), 0.0)
        m_new = np.maximum(m, m_c)
        ref = np.where(np.isfinite(m_new), m_new, 0.0)
        z = np.where(live, z * np.exp(np.where(live, m, 0.0) - ref), 0.0) + np.where(live_c, z_c * np.exp(np.where(live_c, m_c, 0.0) - ref), 0.0)
    return m_new, z


def normalize_rotation_chunks(big_l, weight, n_rot_chunk, p_min=None):
    """The normalisation of `normalize` when the rotations arrive in chunks C_c and only one chunk of
    L is held at a time.  "Only maximal rotational probabilities and sums are necessary":
    sweep 1 carries, per pattern d, the running maximum m_d and the running sum z_d of exp(a - m_d)
    over the chunks seen so far,
        m' = max(m, m_c),   z' = z exp(m - m') + z_c exp(m_c - m'),
    with (m_c, z_c) the max and sum of chunk c alone; sweep 2 revisits every chunk with the final
    (m_d, z_d):  P = exp(a - m_d) / z_d.  Same `p_min` (G20), same s and LL as `normalize`.
    Returns (P float64 [R,N], s float64 [R], LL float)."""
    big_l = np.asarray(big_l).astype(np.float64)
    lw = np.log(np.asarray(weight).astype(np.float64))
    n_rot, n_pat = big_l.shape
    m = np.full(n_pat, -np.inf)
    z = np.zeros(n_pat)
    for r0 in range(0, n_rot, n_rot_chunk):                     # sweep 1
        a = big_l[r0:r0 + n_rot_chunk] + lw[r0:r0 + n_rot_chunk, None]
        m, z = _merge_max_sum(m, z, a)
    p = np.empty_like(big_l)
    for r0 in range(0, n_rot, n_rot_chunk):                     # sweep 2
        a = big_l[r0:r0 + n_rot_chunk] + lw[r0:r0 + n_rot_chunk, None]
        p[r0:r0 + n_rot_chunk] = np.exp(a - m[None, :]) / z[None, :]
    p[p < (P_MIN if p_min is None else p_min)] = 0.0            # G20
    return p, p.sum(axis=1), float((m + np.log(z)).sum())


def iterate_rotation_chunks(model, q, mask, quat, weight, counts, n_rot_chunk, weighted=False, p_min=None):
    """One iteration of Algorithm 1 with the rotation list streamed in chunks of `n_rot_chunk`
    (PAPER.md:164-166): nothing of size R x N or R x P is ever held.
      sweep 1, per chunk: expand -> loglik -> merge the chunk's (max, sum) into the running ones
      sweep 2, per chunk: expand -> loglik (again) -> P with the final (max, sum) -> update -> the
               chunk's contribution to the numerator and denominator grids of Compress
      last: model' = num / den (division as the final step).
    Stage boundaries carry float32 as in `iterate`.  Returns dict(model, s, LL, den)."""
    counts = np.asarray(counts)
    quat = np.asarray(quat, dtype=np.float32)
    weight = np.asarray(weight, dtype=np.float32)
    n = np.asarray(model).shape[0]
    n_rot, n_pat = quat.shape[0], counts.shape[0]
    lw = np.log(weight.astype(np.float64))
    m = np.full(n_pat, -np.inf)
    z = np.zeros(n_pat)
    for r0 in range(0, n_rot, n_rot_chunk):                     # sweep 1
        sl = slice(r0, min(n_rot, r0 + n_rot_chunk))
        w, idx = expand(model, q, quat[sl])
        l32 = loglik(w, idx, counts, mask)[0].astype(np.float32)
        a = l32.astype(np.float64) + lw[sl, None]
        m, z = _merge_max_sum(m, z, a)
    g = n * n * n
    num, den = np.zeros(g), np.zeros(g)
    s_all = np.zeros(n_rot)
    for r0 in range(0, n_rot, n_rot_chunk):                     # sweep 2
        sl = slice(r0, min(n_rot, r0 + n_rot_chunk))
        w, idx = expand(model, q, quat[sl])
        l32 = loglik(w, idx, counts, mask)[0].astype(np.float32)
        a = l32.astype(np.float64) + lw[sl, None]
        p = np.exp(a - m[None, :]) / z[None, :]
        p[p < (P_MIN if p_min is None else p_min)] = 0.0        # G20
        p32 = p.astype(np.float32)
        wn, s = update(p32, counts, mask)
        s_all[sl] = s
        om = s.astype(np.float32) if weighted else (s > 0).astype(np.float32)
        _, num_c, den_c = compress(wn, q, quat[sl], mask, n, slice_w=om)
        num += num_c
        den += den_c
    with np.errstate(divide="ignore", invalid="ignore"):
        new_model = np.where(den > 0, num / den, 0.0)
    return dict(model=new_model.astype(np.float32).reshape(n, n, n), s=s_all, LL=float((m + np.log(z)).sum()), den=den)


# ----------------------------------------------------------------------------------------------
# Adaptive EMC, PAPER.md:205-210 (section 3.4, eq. 3.1)
# ----------------------------------------------------------------------------------------------

def refine_criterion(ll_prev, ll_cur, threshold=0.01):
    """Eq. (3.1): the rotational discretisation is refined when |L^n - L^(n-1)| <= 0.01 |L^n|."""
    return abs(ll_cur - ll_prev) <= threshold * abs(ll_cur)


def refine(model, q, mask, levels, counts, n_iter, threshold=0.01, weighted=False):
    """Adaptive EMC: start on the coarsest rotation list `levels[0]` = (quat, weight) and
    move to the next list "whenever the current value seems too small to improve the likelihood any further",
    i.e. after an iteration n >= 1 whose log-likelihood satisfies eq. (3.1) against iteration n - 1 (the paper
    increases d of eq. (2.7) by one; here the lists are given, DESIGN.md NEXT-1).  The last list is kept.
    Returns dict(model, LL [n_iter], level [n_iter] = index of the list iteration n ran on)."""
    level = 0
    lls, used = [], []
    cur = np.asarray(model, dtype=np.float32)
    for n in range(n_iter):
        quat, weight = levels[level]
        out = iterate(cur, q, mask, quat, weight, counts, weighted=weighted)
        cur = out["model"]
        lls.append(out["LL"])
        used.append(level)
        if n >= 1 and level + 1 < len(levels) and refine_criterion(lls[n - 1], lls[n], threshold):
            level += 1
    return dict(model=cur, LL=np.array(lls), level=np.array(used, dtype=np.int32))


# ----------------------------------------------------------------------------------------------
# The paper's own likelihood: Gaussian with a fluence per (rotation, frame), eqs. (2.2), (2.3),
# (2.5), (2.6), (2.11), PAPER.md:70-89, 124-130  (NEXT-3, readings GA1-GA7)
# ----------------------------------------------------------------------------------------------

def fluence(w, counts, mask):
    """phi[r,d] = sum_i K[d,i]^2 / sum_i W[r,i] K[d,i] over unmasked pixels   (eq. 2.6).
    Where the denominator is 0 (a frame without photons on the slice's support) phi is +inf: K/phi = 0 (GA3).
    Returns float64 [R,N]."""
    use = _use(mask, np.asarray(w).shape[1])
    wd = np.asarray(w, dtype=np.float32).astype(np.float64)[:, use]
    k = np.asarray(counts)[:, use].astype(np.float64)
    num = (k * k).sum(axis=1)                                    # [N]
    den = wd @ k.T                                               # [R,N]
    with np.errstate(divide="ignore", invalid="ignore"):
        return np.where(den > 0, num[None, :] / den, np.inf)


def gaussian_loglik(w, counts, mask, phi, sigma, chunk=8):
    """Q[r,d] = sum_i -(K[d,i]/phi[r,d] - W[r,i])^2 / (2 sigma^2) over unmasked pixels, evaluated term by term as
    eqs. (2.2)-(2.3) print it.  Also returns the scale the tolerance refers to,
    A[r,d] = sum_i ((K/phi)^2 + W^2) / (2 sigma^2).  Returns (Q, A) float64 [R,N]."""
    use = _use(mask, np.asarray(w).shape[1])
    wd = np.asarray(w, dtype=np.float32).astype(np.float64)[:, use]
    k = np.asarray(counts)[:, use].astype(np.float64)
    n_rot, n_pat = wd.shape[0], k.shape[0]
    q = np.empty((n_rot, n_pat))
    a = np.empty((n_rot, n_pat))
    inv = 1.0 / (2.0 * float(sigma) ** 2)
    for r0 in range(0, n_rot, chunk):
        r1 = min(n_rot, r0 + chunk)
        scaled = k[None, :, :] / phi[r0:r1, :, None]             # [r,N,Pu]; K / inf = 0
        diff = scaled - wd[r0:r1, None, :]
        q[r0:r1] = -(diff * diff).sum(axis=2) * inv
        a[r0:r1] = ((scaled * scaled).sum(axis=2) + (wd[r0:r1] ** 2).sum(axis=1)[:, None]) * inv
    return q, a


def update_gaussian(p, counts, mask, phi):
    """W'[r,i] = sum_d P[r,d] K[d,i] / phi[r,d]  /  sum_d P[r,d]   (eq. 2.5 with the index typo read as P_jk, G10;
    numerator = eq. 2.11).  Masked pixels and rows with s[r] = 0 give 0.  Returns (W' float32 [R,P], s float64)."""
    pd = np.asarray(p).astype(np.float64)
    k = np.asarray(counts)
    use = _use(mask, k.shape[1])
    s = pd.sum(axis=1)
    with np.errstate(divide="ignore"):
        num = (pd / phi) @ np.where(use[None, :], k, 0).astype(np.float64)
    with np.errstate(divide="ignore", invalid="ignore"):
        wn = np.where(s[:, None] > 0, num / s[:, None], 0.0)
    wn[:, ~use] = 0.0
    return wn.astype(np.float32), s


def iterate_gaussian(model, q, mask, quat, weight, counts, sigma, weighted=True):
    """One EMC iteration with the paper's Gaussian model: expand (2.9) -> fluence (2.6) from the expanded slices
    -> E-step (2.2)-(2.4) -> M-step (2.5)/(2.11) with the same fluence -> compress (2.12) (or (2.10) with
    weighted=False).  GA1: the fluence is recomputed from the current slices in every iteration and used in the E-
    and M-step of that iteration.  Stage boundaries carry float32 (W, Q, P, W').
    Returns dict(model, W, idx, phi, L, A, P, s, Wn, LL, den)."""
    counts = np.asarray(counts)
    n = np.asarray(model).shape[0]
    w, idx = expand(model, q, quat)
    phi = fluence(w, counts, mask)
    big_q, big_a = gaussian_loglik(w, counts, mask, phi, sigma)
    l32 = big_q.astype(np.float32)
    p, _, ll = normalize(l32, weight)
    p32 = p.astype(np.float32)
    wn, s = update_gaussian(p32, counts, mask, phi)
    om = s.astype(np.float32) if weighted else (s > 0).astype(np.float32)
    new_model, _, den = compress(wn, q, quat, mask, n, slice_w=om)
    return dict(model=new_model, W=w, idx=idx, phi=phi, L=l32, A=big_a, P=p32, s=s, Wn=wn, LL=ll, den=den)

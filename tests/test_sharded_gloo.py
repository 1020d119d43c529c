"""Rotation-sharded iteration (paper_1409_4256_b200/parallel.py) on CPU: world_size 2, gloo.
The three device phases of a rank are supplied by an ORACLE-backed backend defined here (tests may import the oracle;
the product module never does), so what is exercised is the module's own logic: the shares of the rotation list, the
all-gather of the per-pattern statistics in rank order, the all-reduce of the numerator / denominator grids, and that
every rank ends with the same model and log-likelihood as the unsharded oracle iteration."""
import os
import pathlib
import sys

import numpy as np
import torch
import torch.multiprocessing as mp

ROOT = pathlib.Path(__file__).resolve().parents[1]


class OracleBackend:
    """stats / update / finish of one rank with oracle arithmetic (numpy), tensors in and out."""

    def __init__(self):
        self.l32 = None

    def stats(self, model, q, mask, quat, weight, counts, n_rot_total):
        from oracle import emc_oracle as o

        w, idx = o.expand(model.numpy(), q.numpy(), quat.numpy())
        self.l32 = o.loglik(w, idx, counts.numpy(), mask.numpy())[0].astype(np.float32)
        self.lw = np.log(weight.numpy().astype(np.float64))
        a = self.l32.astype(np.float64) + self.lw[:, None]
        top = a.argmax(axis=0)
        cols = np.arange(a.shape[1])
        z = np.exp(a - a[top, cols][None, :]).sum(axis=0)
        return torch.from_numpy(np.stack([self.l32[top, cols].astype(np.float64), self.lw[top], z]).astype(np.float32))

    def update(self, model, q, mask, quat, weight, counts, n_rot_total, stats_all):
        from oracle import emc_oracle as o

        st = stats_all.numpy().astype(np.float64)                  # [world, 3, N]
        key = st[:, 0] + st[:, 1]
        m = key.max(axis=0)
        z = (st[:, 2] * np.exp(key - m[None, :])).sum(axis=0)
        a = self.l32.astype(np.float64) + self.lw[:, None]
        p = np.exp(a - m[None, :]) / z[None, :]
        p[p < o.P_MIN] = 0.0                                       # the oracle's default: nothing flushed (G20)
        wn, s = o.update(p.astype(np.float32), counts.numpy(), mask.numpy())
        n = model.shape[0]
        _, num, den = o.compress(wn, q.numpy(), quat.numpy(), mask.numpy(), n, slice_w=(s > 0).astype(np.float32))
        ll = float((m + np.log(z)).sum())
        return (torch.from_numpy(np.stack([num, den]).reshape(2, n, n, n)), torch.tensor([ll], dtype=torch.float64),
                torch.from_numpy(s))

    def finish(self, numden):
        num, den = numden[0].numpy(), numden[1].numpy()
        with np.errstate(divide="ignore", invalid="ignore"):
            return torch.from_numpy(np.where(den > 0, num / den, 0.0).astype(np.float32))


def _worker(rank, world, port, out):
    import torch.distributed as dist

    sys.path.insert(0, str(ROOT))
    from emc_inputs import make_inputs
    from paper_1409_4256_b200 import parallel

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    inp = make_inputs("T0")
    t = lambda x: torch.from_numpy(np.ascontiguousarray(x))
    res = parallel.iterate_sharded(t(inp.model_init), t(inp.q), t(inp.mask), t(inp.quat[0]), t(inp.weight[0]), t(inp.counts),
                                   n_iter=2, backend=OracleBackend())
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, res["model"].numpy(), res["loglik"].numpy(), res["s"].numpy(), res["bounds"]))


def test_shard_bounds_cover_the_list():
    sys.path.insert(0, str(ROOT))
    from paper_1409_4256_b200.parallel import shard_bounds

    for n_rot, world in [(60, 2), (61, 4), (7, 7), (25000, 8)]:
        b = [shard_bounds(n_rot, world, r) for r in range(world)]
        assert b[0][0] == 0 and b[-1][1] == n_rot
        assert all(b[i][1] == b[i + 1][0] for i in range(world - 1))
        sizes = [r1 - r0 for r0, r1 in b]
        assert max(sizes) - min(sizes) <= 1


def test_two_ranks_reproduce_the_unsharded_iteration():
    sys.path.insert(0, str(ROOT))
    from emc_inputs import make_inputs
    from oracle import emc_oracle as o

    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted((out.get(timeout=300) for _ in procs), key=lambda x: x[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    inp = make_inputs("T0")
    m, ref = inp.model_init, None
    lls = []
    for _ in range(2):
        ref = o.iterate(m, inp.q, inp.mask, inp.quat[0], inp.weight[0], inp.counts)
        m = ref["model"]
        lls.append(ref["LL"])
    (r0, m0, ll0, s0, b0), (r1, m1, ll1, s1, b1) = got
    assert np.array_equal(m0, m1) and np.array_equal(ll0, ll1)          # every rank holds the same result
    assert b0 == (0, 30) and b1 == (30, 60)
    assert np.allclose(ll0, lls, rtol=1e-6)
    scale = np.abs(ref["model"]).max()
    assert np.abs(m0 - ref["model"]).max() <= 1e-4 * scale
    s_all = np.concatenate([s0, s1])
    assert np.abs(s_all - ref["s"]).max() <= 1e-4 * max(1.0, ref["s"].max())

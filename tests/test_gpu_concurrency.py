"""Two workspaces, two contexts, two streams, two host threads at once (`-m gpu`): libemc keeps no process-wide CUDA
state (include/emc.h conventions), so concurrent calls with host-resident patterns and per-stage timing must give
what the same calls give one after the other."""
import threading

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

emc = pytest.importorskip("paper_1409_4256_b200")


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def test_two_streams_two_contexts(inputs_cache):
    cases = [inputs_cache("T1", n_pat=4200), inputs_cache("T2")]
    flags = emc.EMC_PATTERNS_ON_HOST | emc.EMC_PROFILE_STAGES
    jobs = []
    for inp in cases:
        s = len(inp.quat) - 1
        jobs.append(dict(args=(dev(inp.model_init), dev(inp.q), dev(inp.mask), dev(inp.quat[s]), dev(inp.weight[s])),
                         pinned=torch.from_numpy(inp.counts.copy()).pin_memory(),
                         chunk=0 if inp.cfg.name == "T1" else 200, ctx=emc.EmcContext(), stream=torch.cuda.Stream()))
    torch.cuda.synchronize()

    def run(job, n_rep, out):
        with torch.cuda.stream(job["stream"]):
            for _ in range(n_rep):
                r = emc.emc_iterate(*job["args"], job["pinned"], n_iter=2, n_pat_chunk=job["chunk"], flags=flags,
                                    ctx=job["ctx"], ws=out.get("ws"))
                out["ws"] = r["ws"]
            out["model"], out["ll"] = r["model"], r["loglik"]
            job["stream"].synchronize()

    serial = [dict(), dict()]
    for j, o_ in zip(jobs, serial):
        run(j, 1, o_)
    for j in jobs:
        emc.emc_profile_read(j["ctx"])
    both = [dict(ws=serial[0]["ws"]), dict(ws=serial[1]["ws"])]
    threads = [threading.Thread(target=run, args=(j, 6, o_)) for j, o_ in zip(jobs, both)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    for j, a, b in zip(jobs, serial, both):
        ma, mb = a["model"].cpu().numpy(), b["model"].cpu().numpy()
        assert np.abs(ma - mb).max() <= 1e-3 * np.abs(ma).max()           # fp32 atomics order the second iteration
        assert np.allclose(a["ll"].cpu().numpy(), b["ll"].cpu().numpy(), rtol=1e-6)
        prof = emc.emc_profile_read(j["ctx"])
        # log-likelihood launches per call: T1 = 3 sub-ranges of the pipelined first iteration + 1; T2 = 2 x 3 chunks
        assert prof["loglik"][1] == 6 * ((3 + 1) if j["chunk"] == 0 else 2 * 3)
        assert all(v[0] >= 0 for v in prof.values())
        with torch.cuda.stream(j["stream"]):
            emc.emc_check(b["ws"])
        j["ctx"].close()

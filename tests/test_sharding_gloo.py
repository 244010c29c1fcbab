"""N > 1 path on CPU: world_size-2 (and 3) gloo processes shard the centres of C1s / C4s, each computes its rows with
the ORACLE (no GPU here), exchanges g_r through paper_2504_16068_b200.sharding.ShardedForces and gathers its own
forces; the concatenation must equal the single-process oracle forces and energy."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.join(ROOT, "tests")):
    if p not in sys.path:
        sys.path.insert(0, p)


def test_partition_balanced_and_covering():
    from paper_2504_16068_b200.sharding import partition_centres
    rng = np.random.default_rng(0)
    for world in (1, 2, 3, 8):
        for N in (1, 5, 64, 1000):
            deg = rng.integers(0, 40, size=N)
            rp = np.concatenate([[0], np.cumsum(deg)]).astype(np.int32)
            parts = partition_centres(rp, world)
            assert len(parts) == world and parts[0][0] == 0 and parts[-1][1] == N
            assert all(parts[r][1] == parts[r + 1][0] for r in range(world - 1))
            assert all(a <= b for a, b in parts)
            if N >= 100:
                edges = [int(rp[b] - rp[a]) for a, b in parts]
                assert max(edges) <= rp[-1] / world + 40          # within one row of perfectly balanced


def _worker(rank, world, port, name, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import _chain
    import oracle as orc
    from paper_2504_16068_b200.sharding import ShardedForces
    from workloads.inputs import sub_inputs
    inp = _chain.make_inputs(name)

    def compute(c_lo, c_hi):
        if c_hi == c_lo:
            return torch.zeros((0, 3), dtype=torch.float64), torch.zeros((), dtype=torch.float64)
        sub = sub_inputs(inp, c_lo, c_hi)
        r = _chain.oracle_chain(sub, want_gw=False, forces=False)
        return torch.from_numpy(r["g_r"]), torch.tensor(float(np.sum(r["e_edge"])), dtype=torch.float64)

    def gather(rp_slice, rev, g_all):
        return torch.from_numpy(orc.force_gather(rp_slice, rev, g_all.numpy()))

    sh = ShardedForces(inp["row_ptr"], inp["rev"], compute, gather)
    F_loc, e_tot, (c_lo, c_hi) = sh.run()
    q.put((rank, c_lo, c_hi, F_loc.numpy(), float(e_tot.item())))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("name,world", [("C1s", 2), ("C4s", 3)])
def test_sharded_forces_match_single_process(name, world):
    import _chain
    inp = _chain.make_inputs(name)
    ref = _chain.oracle_chain(inp, want_gw=False)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, world, port, name, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = [q.get(timeout=300) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    F = np.zeros_like(ref["F"])
    for rank, c_lo, c_hi, F_loc, e_tot in got:
        F[c_lo:c_hi] = F_loc
        assert abs(e_tot - float(np.sum(ref["e_edge"]))) <= 1e-9 * abs(float(np.sum(ref["e_edge"])))
    assert np.max(np.abs(F - ref["F"])) <= 1e-12 * np.max(np.abs(ref["F"]))

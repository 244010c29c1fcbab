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


def test_halo_plan_index_lists():
    """HaloPlan without any process group: for every rank of worlds 1..5 the extended array [own rows ; received rows] indexed by
    rev_loc reproduces g_r[rev[e]] for every own edge, and the two sides of every rank pair agree on count and order"""
    import _chain
    from paper_2504_16068_b200.sharding import HaloPlan
    inp = _chain.make_inputs("C4s")
    rp, rev = inp["row_ptr"], inp["rev"]
    E = int(rp[-1])
    g = np.arange(3 * E, dtype=np.float64).reshape(E, 3)            # row e identifies global edge e
    for world in (1, 2, 3, 5):
        plans = [HaloPlan(rp, rev, world, r) for r in range(world)]
        for r, pr in enumerate(plans):
            ext = np.full((pr.n_local + pr.n_halo, 3), -1.0)
            ext[:pr.n_local] = g[pr.e0:pr.e1]
            for s_, ps in enumerate(plans):
                if s_ == r:
                    continue
                rows = g[ps.e0 + ps.send_idx[r]]                     # what s sends to r, in s's order
                assert rows.shape[0] == pr.recv_cnt[s_]
                ext[pr.recv_off[s_]:pr.recv_off[s_] + pr.recv_cnt[s_]] = rows
            assert np.array_equal(ext[pr.rev_loc], g[rev[pr.e0:pr.e1]])
            assert pr.row_ptr_loc[0] == 0 and pr.row_ptr_loc[-1] == pr.n_local
        assert sum(pr.n_local for pr in plans) == E


def _worker(rank, world, port, name, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import _chain
    import oracle as orc
    from paper_2504_16068_b200.sharding import ShardedForces
    from workloads.inputs import sub_inputs
    inp = _chain.make_inputs(name)
    sh = ShardedForces(inp["row_ptr"], inp["rev"], device="cpu", dtype=torch.float64)
    hp = sh.plan
    # (1) stub compute: row e of g_r names global edge e; after the exchange every own edge must see its reverse's row
    sh.g_local.copy_(torch.arange(3 * hp.e0, 3 * hp.e1, dtype=torch.float64).reshape(-1, 3))
    sh.exchange()
    want = np.arange(3 * int(inp["row_ptr"][-1]), dtype=np.float64).reshape(-1, 3)[inp["rev"][hp.e0:hp.e1]]
    stub_ok = bool(np.array_equal(sh.g_ext.numpy()[hp.rev_loc], want))
    # (2) the oracle as the compute on the rank's centres
    if hp.c_hi > hp.c_lo:
        r = _chain.oracle_chain(sub_inputs(inp, hp.c_lo, hp.c_hi), want_gw=False, forces=False)
        sh.g_local.copy_(torch.from_numpy(r["g_r"]))
        e_loc = torch.tensor([float(np.sum(r["e_edge"]))], dtype=torch.float64)
    else:
        e_loc = torch.zeros(1, dtype=torch.float64)
    sh.exchange()
    F_loc = orc.force_gather(hp.row_ptr_loc, hp.rev_loc, sh.g_ext.numpy())
    e_tot = sh.reduce_sum(e_loc)
    F_all = sh.gather_forces(torch.from_numpy(F_loc), inp["N"])
    q.put((rank, hp.c_lo, hp.c_hi, F_loc, float(e_tot.item()), stub_ok, F_all.numpy(), sh.halo_bytes))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("name,world", [("C1s", 2), ("C4s", 3)])
def test_sharded_forces_match_single_process(name, world):
    """world_size-2 / 3 gloo processes: halo exchange of the cut edges' g_r rows, forces gathered by the owners.  The owners'
    forces are BITWISE the single-process oracle's (same per-atom order, same operands); the energy is a sum over ranks."""
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
    for rank, c_lo, c_hi, F_loc, e_tot, stub_ok, F_all, halo_bytes in got:
        assert stub_ok
        F[c_lo:c_hi] = F_loc
        assert abs(e_tot - float(np.sum(ref["e_edge"]))) <= 1e-9 * abs(float(np.sum(ref["e_edge"])))
        assert np.array_equal(F_all, ref["F"])
        assert halo_bytes > 0
    assert np.array_equal(F, ref["F"])

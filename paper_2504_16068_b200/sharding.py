"""Multi-GPU host logic: Allegro is strictly local, E_tot = sum_i eps_i(edges of centre i), so the
path shards by CENTRE ATOM with no data-path collective in the forward pass or in the tensor-product / embedding
VJPs.  The one exchange is the force assembly: atom a needs g_r of the reverse edges of its row, which other ranks
own.  Here every rank all-gathers the per-edge gradients g_r[E,3] (12 bytes per edge: 4.4 MB at C1, 35 MB at C2;
latency-bound over NVLink/NVSwitch) and then gathers the forces of ITS OWN atoms with the deterministic CSR
force_gather (no scatter-add, no float atomics), as a spatial-decomposition MD code keeps forces with the owner.

The compute itself is injected (`compute_g_r`): on a GPU box it is the library's kernels on the rank's rows, in the
CPU tests it is the oracle; only the partition, the padding and the collective live here.
"""
import numpy as np
import torch
import torch.distributed as dist


def partition_centres(row_ptr, world):
    """contiguous centre ranges [(c_lo, c_hi)] * world, balanced by edge count (rank r gets the centres whose
    first edge falls in [r E / world, (r+1) E / world)); ranges may be empty"""
    rp = np.asarray(row_ptr, dtype=np.int64)
    N, E = rp.shape[0] - 1, int(rp[-1])
    cuts = [int(np.searchsorted(rp[:-1], (r * E + world - 1) // world, side="left")) for r in range(world)] + [N]
    cuts[0] = 0
    return [(cuts[r], cuts[r + 1]) for r in range(world)]


class ShardedForces:
    """rank-local piece of one MD step: run compute_g_r on the rank's centres, exchange g_r, gather own forces.

    compute_g_r(c_lo, c_hi) -> (g_r_local [E_local, 3] tensor, energy_local 0-d tensor)
    force_gather(row_ptr_slice, rev, g_r_all) -> F_local [c_hi - c_lo, 3] tensor   (row_ptr_slice keeps GLOBAL edge offsets)
    """

    def __init__(self, row_ptr, rev, compute_g_r, force_gather, group=None):
        self.group = group
        self.world, self.rank = dist.get_world_size(group), dist.get_rank(group)
        self.row_ptr = np.asarray(row_ptr, dtype=np.int32)
        self.rev = rev
        self.parts = partition_centres(self.row_ptr, self.world)
        self.edge_ranges = [(int(self.row_ptr[a]), int(self.row_ptr[b])) for a, b in self.parts]
        self.pad = max(e1 - e0 for e0, e1 in self.edge_ranges)
        self.compute_g_r, self.force_gather = compute_g_r, force_gather

    def run(self):
        c_lo, c_hi = self.parts[self.rank]
        g_loc, e_loc = self.compute_g_r(c_lo, c_hi)
        buf = torch.zeros((self.pad, 3), dtype=g_loc.dtype, device=g_loc.device)
        buf[: g_loc.shape[0]] = g_loc
        gathered = [torch.empty_like(buf) for _ in range(self.world)]
        dist.all_gather(gathered, buf, group=self.group)
        g_all = torch.cat([gathered[r][: e1 - e0] for r, (e0, e1) in enumerate(self.edge_ranges)], dim=0)
        e_tot = e_loc.clone().reshape(1)
        dist.all_reduce(e_tot, op=dist.ReduceOp.SUM, group=self.group)
        F_loc = self.force_gather(self.row_ptr[c_lo:c_hi + 1], self.rev, g_all)
        return F_loc, e_tot, (c_lo, c_hi)

"""The single-layer chain of the scalar-weight configs as a sequence of library calls (marshalling only).

    w = radial(r)  ->  Eenv = env_embed(w)  ->  out = tp_forward(V, Eenv, path_w)
    -> e_edge, G = edge_energy(out, q, kappa)  ->  gV, gEenv, g_path_w = tp_backward(G, ...)
    -> g_r, g_w = env_embed_backward(gEenv)  ->  g_r += radial_backward(g_w)  ->  F = force_gather(g_r)
    (molecule batches: E_mol = segment_sum over the edges of each molecule's centres)

This is one "MD step" for one tensor-product layer: positions (as edge vectors) in, energy and forces out.
"""
import numpy as np
import torch

import paper_2504_16068_b200 as ab


def to_device(inp, device="cuda"):
    d = {}
    for k in ("row_ptr", "rev", "rvec", "V", "W_r", "path_w", "q", "edge_mol_ptr"):
        v = inp.get(k)
        if v is not None:
            d[k] = v.to(device) if torch.is_tensor(v) else torch.from_numpy(np.ascontiguousarray(v)).to(device)
    return d


def gpu_chain(inp, dev=None, items=None, want_gw=True, plan=None):
    """The same chain through the C ABI.  Returns torch tensors on the device."""
    if dev is None:
        dev = to_device(inp)
    if plan is None:
        plan = ab.Plan(inp["lmax"], inp["n"], ab.F64 if inp["dt"] == np.float64 else ab.F32, ab.W_SCALAR)
    it = None if items is None else torch.from_numpy(np.ascontiguousarray(items)).to("cuda")
    rp, rvec, V, pw = dev["row_ptr"], dev["rvec"], dev["V"], dev["path_w"]
    w = ab.radial_forward(rvec, dev["W_r"], inp["rc"])
    Eenv = ab.env_embed(plan, rp, rvec, w, inp["scale"], items=it)
    out = ab.tp_forward(plan, rp, V, Eenv, pw, items=it)
    e_edge, G = ab.edge_energy(plan, out, dev["q"], inp["kappa"])
    gV, gE, gpw = ab.tp_backward(plan, rp, G, V, Eenv, pw, items=it, want_gV=True, want_g_path_w=want_gw)
    g_r, g_w = ab.env_embed_backward(plan, rp, gE, rvec, w, inp["scale"])
    g_r_env = g_r.clone()
    ab.radial_backward(rvec, dev["W_r"], inp["rc"], g_w, g_r)
    F = ab.force_gather(rp, dev["rev"], g_r)
    res = dict(w=w, Eenv=Eenv, out=out, e_edge=e_edge, G=G, gV=gV, gEenv=gE, g_path_w=gpw, g_w=g_w, g_r_env=g_r_env, g_r=g_r, F=F)
    if dev.get("edge_mol_ptr") is not None:
        res["E_mol"] = ab.segment_sum(dev["edge_mol_ptr"], e_edge)
    return res


class SingleLayerStep:
    """One MD step of one tensor-product layer with every buffer allocated once (nothing is allocated and no
    host synchronisation happens inside run()): the object bench.py times.  `want_gV` selects the full VJP
    (dE/dV as well, what a layer inside a deeper network needs) or the force-only VJP.  `mode`:
      "separate" : tp_forward -> edge_energy -> tp_backward                     (out, G both cross HBM twice)
      "epilogue" : tp_forward_energy (out, e_edge, G from one kernel) -> tp_backward
      "onthefly" : tp_forward_energy (out, e_edge) -> tp_backward_energy (cotangent formed from out in registers;
                   G never exists in HBM)
      "fused"    : tp_fused_energy: forward, energy and VJP in ONE kernel (V read once, gV written once, out and G never
                   exist in HBM; self.out stays unwritten)
    `fused_geometry`: env_radial_forward / env_radial_backward (w and g_w never exist in HBM) instead of
    radial_forward + env_embed / env_embed_backward + radial_backward."""

    def __init__(self, plan, dev, rc, kappa, scale=1.0, want_gV=True, want_g_path_w=False, items=None, mode="onthefly", fused_geometry=True,
                 sharded=None):
        """sharded: a sharding.ShardedForces when `dev` holds ONE RANK'S rows of a system split over several GPUs (row_ptr / rev are the
        rank-local index arrays of its HaloPlan): g_r is written into its extended array, the halo exchange runs before the force
        gather, energies (and g_path_w) are summed over the ranks"""
        assert mode in ("separate", "epilogue", "onthefly", "fused")
        self.sharded = sharded
        self.plan, self.dev, self.rc, self.kappa, self.scale, self.mode = plan, dev, rc, kappa, scale, mode
        self.fused_geometry = fused_geometry
        rp, rvec, V = dev["row_ptr"], dev["rvec"], dev["V"]
        self.N, self.E = rp.shape[0] - 1, rvec.shape[0]
        self.items = items
        dt, dv = rvec.dtype, rvec.device
        n = plan.n
        self.w = None if fused_geometry else torch.empty((self.E, n), dtype=dt, device=dv)
        self.Eenv = torch.empty((self.N, n, plan.dE), dtype=dt, device=dv)
        self.out = torch.empty_like(V) if mode != "fused" else None
        self.e_edge = torch.empty((self.E,), dtype=dt, device=dv)
        self.G = torch.empty_like(V) if mode in ("separate", "epilogue") else None
        self.gV = torch.empty_like(V) if want_gV else None
        self.gEenv = torch.empty_like(self.Eenv)
        self.g_path_w = torch.empty((plan.P,), dtype=dt, device=dv) if want_g_path_w else None
        self.g_r = torch.empty_like(rvec) if sharded is None else sharded.g_local
        self.g_w = None if fused_geometry else torch.empty_like(self.w)
        self.F = torch.empty((self.N, 3), dtype=dt, device=dv)
        self.e_tot = torch.empty((1,), dtype=dt, device=dv)
        self.e_ptr = torch.tensor([0, self.E], dtype=torch.int32, device=dv)
        self.ws_env = torch.empty(max(ab.env_workspace(plan, self.N, items), 16), dtype=torch.uint8, device=dv)
        self.ws_bwd = torch.empty(max(ab.tp_backward_workspace(plan, self.N, self.E, items, want_g_path_w), 16), dtype=torch.uint8, device=dv)
        self.marks = None      # optional list of (name, start_event, end_event) filled by run(mark=True)
        self.bind_weights()

    def bind_weights(self):
        """fold dev["path_w"] into the plan's combined tensor (once: MD weights are fixed; call again after changing them)"""
        self.plan.bind_weights(self.dev["path_w"])

    def run(self, mark=False):
        p, d, it = self.plan, self.dev, self.items
        rp, rvec, V, pw = d["row_ptr"], d["rvec"], d["V"], None      # path weights: the table bound to the plan
        ev = []

        def timed(name, fn):
            if not mark:
                return fn()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            r = fn()
            b.record()
            ev.append((name, a, b))
            return r

        bw = dict(items=it, want_gV=self.gV is not None, gV=self.gV, gEenv=self.gEenv, g_path_w=self.g_path_w, workspace=self.ws_bwd)
        if self.fused_geometry:
            timed("env_radial_forward", lambda: ab.env_radial_forward(p, rp, rvec, d["W_r"], self.rc, self.scale, items=it, Eenv=self.Eenv,
                                                                      workspace=self.ws_env))
        else:
            timed("radial_forward", lambda: ab.radial_forward(rvec, d["W_r"], self.rc, w=self.w))
            timed("env_embed", lambda: ab.env_embed(p, rp, rvec, self.w, self.scale, items=it, Eenv=self.Eenv, workspace=self.ws_env))
        if self.mode == "separate":
            timed("tp_forward", lambda: ab.tp_forward(p, rp, V, self.Eenv, pw, items=it, out=self.out))
            timed("edge_energy", lambda: ab.edge_energy(p, self.out, d["q"], self.kappa, e_edge=self.e_edge, G=self.G))
            timed("tp_backward", lambda: ab.tp_backward(p, rp, self.G, V, self.Eenv, pw, **bw))
        elif self.mode == "epilogue":
            timed("tp_forward_energy", lambda: ab.tp_forward_energy(p, rp, V, self.Eenv, pw, d["q"], self.kappa, items=it, out=self.out,
                                                                    e_edge=self.e_edge, G=self.G))
            timed("tp_backward", lambda: ab.tp_backward(p, rp, self.G, V, self.Eenv, pw, **bw))
        elif self.mode == "onthefly":
            timed("tp_forward_energy", lambda: ab.tp_forward_energy(p, rp, V, self.Eenv, pw, d["q"], self.kappa, items=it, out=self.out,
                                                                    e_edge=self.e_edge, want_G=False))
            timed("tp_backward_energy", lambda: ab.tp_backward_energy(p, rp, self.out, V, self.Eenv, pw, d["q"], self.kappa, **bw))
        else:
            timed("tp_fused_energy", lambda: ab.tp_fused_energy(p, rp, V, self.Eenv, pw, d["q"], self.kappa, e_edge=self.e_edge, **bw))
        if self.fused_geometry:
            timed("env_radial_backward", lambda: ab.env_radial_backward(p, rp, self.gEenv, rvec, d["W_r"], self.rc, self.scale, g_rvec=self.g_r))
        else:
            timed("env_embed_backward", lambda: ab.env_embed_backward(p, rp, self.gEenv, rvec, self.w, self.scale, g_rvec=self.g_r, g_w=self.g_w))
            timed("radial_backward", lambda: ab.radial_backward(rvec, d["W_r"], self.rc, self.g_w, self.g_r))
        if self.sharded is None:
            timed("force_gather", lambda: ab.force_gather(rp, d["rev"], self.g_r, F=self.F))
            timed("segment_sum", lambda: ab.segment_sum(self.e_ptr, self.e_edge, out=self.e_tot))
        else:
            timed("halo_exchange", self.sharded.exchange)
            timed("force_gather", lambda: ab.force_gather(rp, d["rev"], self.sharded.g_ext, F=self.F))
            timed("segment_sum", lambda: ab.segment_sum(self.e_ptr, self.e_edge, out=self.e_tot))
            timed("energy_all_reduce", lambda: self.sharded.reduce_sum(self.e_tot))
            if self.g_path_w is not None:
                self.sharded.reduce_sum(self.g_path_w)
        if mark:
            self.marks = ev
        return self.F, self.e_tot

    def run_forward(self):
        """forward only (BASELINE.json:configs[1]: "forward only, then forward+force VJP"): embedding, tensor product with the
        energy epilogue, energy sum"""
        p, d, it = self.plan, self.dev, self.items
        rp, rvec, V = d["row_ptr"], d["rvec"], d["V"]
        if self.fused_geometry:
            ab.env_radial_forward(p, rp, rvec, d["W_r"], self.rc, self.scale, items=it, Eenv=self.Eenv, workspace=self.ws_env)
        else:
            ab.radial_forward(rvec, d["W_r"], self.rc, w=self.w)
            ab.env_embed(p, rp, rvec, self.w, self.scale, items=it, Eenv=self.Eenv, workspace=self.ws_env)
        if self.out is None:       # mode "fused" never materialises `out`: the forward-only timing needs a buffer of its own
            self.out = torch.empty_like(V)
        ab.tp_forward_energy(p, rp, V, self.Eenv, None, d["q"], self.kappa, items=it, out=self.out, e_edge=self.e_edge, want_G=False)
        ab.segment_sum(self.e_ptr, self.e_edge, out=self.e_tot)
        return self.e_tot

    def forward_bytes(self):
        b = self.algorithmic_bytes()
        return (b["env_radial_forward"] if self.fused_geometry else b["radial_forward"] + b["env_embed"]) + 2 * self.E * self.plan.n * self.plan.dV * (
            4 if self.plan.dtype == ab.F32 else 8) + b["segment_sum"]

    def algorithmic_bytes(self):
        """HBM bytes each call must move at least once: dict name -> bytes per step"""
        p = self.plan
        s = 4 if p.dtype == ab.F32 else 8
        E, N, n, dV, dE = self.E, self.N, p.n, p.dV, p.dE
        feat, env, wrow = E * n * dV * s, N * n * dE * s, E * n * s
        bwd = (3 if self.gV is not None else 2) * feat + 2 * env + (N + 1) * 4
        return {
            "radial_forward": E * 3 * s + wrow,
            "env_embed": E * 3 * s + wrow + env + (N + 1) * 4,
            "tp_forward": 2 * feat + env + (N + 1) * 4,
            "edge_energy": 2 * feat + E * s,
            "tp_forward_energy": (3 if self.G is not None else 2) * feat + env + E * s + (N + 1) * 4,
            "tp_backward": bwd,
            "tp_backward_energy": bwd,
            "tp_fused_energy": (2 if self.gV is not None else 1) * feat + 2 * env + E * s + (N + 1) * 4,
            "env_radial_forward": E * 3 * s + env + (N + 1) * 4,
            "env_radial_backward": env + 2 * E * 3 * s + (N + 1) * 4,
            "env_embed_backward": env + E * 3 * s + wrow + wrow + E * 3 * s + (N + 1) * 4,
            "radial_backward": E * 3 * s + wrow + 2 * E * 3 * s,
            "force_gather": 2 * E * 3 * s + E * 4 + N * 3 * s + (N + 1) * 4,
            "segment_sum": E * s,
        }


class HostStep:
    """The same step through the C ABI's host entry point allegro_layer_step_host: every input of the step (row_ptr, rev,
    rvec, V and the small parameter tensors) sits in pinned host memory and is copied to the device inside the call;
    forces and the total energy come back to pinned host memory before the call returns."""

    KEYS = ("row_ptr", "rev", "rvec", "V", "W_r", "path_w", "q")

    def __init__(self, step, inp=None):
        self.step = step
        d, p = step.dev, step.plan
        self.host = {k: torch.empty(d[k].shape, dtype=d[k].dtype, pin_memory=True).copy_(d[k]) for k in self.KEYS}
        self.F_host = torch.empty(step.F.shape, dtype=step.F.dtype, pin_memory=True)
        self.e_host = torch.empty(step.e_tot.shape, dtype=step.e_tot.dtype, pin_memory=True)
        self.want_gV = step.gV is not None
        nbytes = ab.layer_step_host_workspace(p, step.N, step.E, d["W_r"].shape[1], self.want_gV)
        self.ws = torch.empty(nbytes, dtype=torch.uint8, device=d["rvec"].device)
        self.h2d_bytes = int(sum(v.numel() * v.element_size() for v in self.host.values()))
        self.d2h_bytes = int(self.F_host.numel() * self.F_host.element_size() + self.e_host.numel() * self.e_host.element_size())

    def run(self):
        h, s = self.host, self.step
        return ab.layer_step_host(s.plan, h["row_ptr"], h["rev"], h["rvec"], h["V"], h["W_r"], s.rc, h["path_w"], h["q"], s.kappa, s.scale,
                                  self.F_host, self.e_host, self.ws, want_gV=self.want_gV)


class ChunkedStep:
    """The same step for a system whose feature tensors do not fit HBM four times (C3: 85.8 GB per tensor): V stays
    resident, the centres are processed in `n_chunks` contiguous ranges that reuse one set of chunk-sized work buffers
    (out, gV), and the per-edge results that the force assembly needs (g_r, e_edge) are written into full-size arrays.
    Chunks are independent because every per-edge / per-centre quantity depends on one centre (strict locality).
    Call sequence per chunk: env_radial_forward -> tp_fused_energy (forward + energy + VJP in one kernel: no `out` buffer at
    all) -> env_radial_backward; then one force_gather and one segment_sum over the whole system.  fused=False keeps the two-kernel
    sequence tp_forward_energy -> tp_backward_energy with a chunk-sized `out` buffer (parity tests read it)."""

    def __init__(self, plan, dev, row_ptr_host, rc, kappa, scale=1.0, n_chunks=8, want_gV=True, fused=None):
        from .sharding import partition_centres
        fused = plan.l_max <= 2 if fused is None else fused      # at l_max = 3 the two-kernel sequence is faster
        self.fused = fused
        self.plan, self.dev, self.rc, self.kappa, self.scale = plan, dev, rc, kappa, scale
        rp_h = np.asarray(row_ptr_host, dtype=np.int64)
        self.N, self.E = rp_h.shape[0] - 1, int(rp_h[-1])
        self.parts = [p for p in partition_centres(rp_h, n_chunks) if p[1] > p[0]]
        dv, dt = dev["rvec"].device, dev["rvec"].dtype
        self.chunks = []
        emax = 0
        for c0, c1 in self.parts:
            e0, e1 = int(rp_h[c0]), int(rp_h[c1])
            rp_c = torch.from_numpy((rp_h[c0:c1 + 1] - e0).astype(np.int32)).to(dv)
            self.chunks.append((c0, c1, e0, e1, rp_c))
            emax = max(emax, e1 - e0)
        n = plan.n
        self.Eenv = torch.empty((self.N, n, plan.dE), dtype=dt, device=dv)
        self.gEenv = torch.empty_like(self.Eenv)
        self.out = None if fused else torch.empty((emax, n, plan.dV), dtype=dt, device=dv)
        self.gV = torch.empty((emax, n, plan.dV), dtype=dt, device=dv) if want_gV else None
        self.e_edge = torch.empty((self.E,), dtype=dt, device=dv)
        self.g_r = torch.empty((self.E, 3), dtype=dt, device=dv)
        self.F = torch.empty((self.N, 3), dtype=dt, device=dv)
        self.e_tot = torch.empty((1,), dtype=dt, device=dv)
        self.e_ptr = torch.tensor([0, self.E], dtype=torch.int32, device=dv)
        self.ws = torch.empty(16, dtype=torch.uint8, device=dv)
        self.emax = emax
        plan.bind_weights(dev["path_w"])

    def run(self, keep=None, mark=False):
        """keep: optional dict chunk_index -> dict that receives clones of that chunk's out / gV (parity tests); a dict with a "rows" entry
        (list of GLOBAL edge ranges (e_lo, e_hi) inside the chunk) receives only those rows, as lists under "out" / "gV";
        mark: record CUDA events around every call -> self.marks = [(name, start, end)] (one entry per call and chunk)"""
        p, d = self.plan, self.dev
        ev = []

        def timed(name, fn):
            if not mark:
                return fn()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            r = fn()
            b.record()
            ev.append((name, a, b))
            return r

        self.marks = ev
        for k, (c0, c1, e0, e1, rp_c) in enumerate(self.chunks):
            m = e1 - e0
            rvec, V = d["rvec"][e0:e1], d["V"][e0:e1]
            Eenv, gE = self.Eenv[c0:c1], self.gEenv[c0:c1]
            out = None if self.out is None else self.out[:m]
            gV = None if self.gV is None else self.gV[:m]
            timed("env_radial_forward", lambda: ab.env_radial_forward(p, rp_c, rvec, d["W_r"], self.rc, self.scale, Eenv=Eenv))
            if self.fused:
                timed("tp_fused_energy", lambda: ab.tp_fused_energy(p, rp_c, V, Eenv, None, d["q"], self.kappa, e_edge=self.e_edge[e0:e1],
                                                                    want_gV=gV is not None, gV=gV, gEenv=gE, workspace=self.ws))
            else:
                timed("tp_forward_energy", lambda: ab.tp_forward_energy(p, rp_c, V, Eenv, None, d["q"], self.kappa, out=out,
                                                                        e_edge=self.e_edge[e0:e1], want_G=False))
                timed("tp_backward_energy", lambda: ab.tp_backward_energy(p, rp_c, out, V, Eenv, None, d["q"], self.kappa,
                                                                          want_gV=gV is not None, gV=gV, gEenv=gE, workspace=self.ws))
            timed("env_radial_backward", lambda: ab.env_radial_backward(p, rp_c, gE, rvec, d["W_r"], self.rc, self.scale,
                                                                        g_rvec=self.g_r[e0:e1]))
            if keep is not None and k in keep:
                if "rows" in keep[k]:
                    keep[k]["out"] = [None if out is None else out[a - e0:b - e0].clone() for a, b in keep[k]["rows"]]
                    keep[k]["gV"] = [None if gV is None else gV[a - e0:b - e0].clone() for a, b in keep[k]["rows"]]
                else:
                    keep[k].update(out=None if out is None else out.clone(), gV=None if gV is None else gV.clone())
        timed("force_gather", lambda: ab.force_gather(d["row_ptr"], d["rev"], self.g_r, F=self.F))
        timed("segment_sum", lambda: ab.segment_sum(self.e_ptr, self.e_edge, out=self.e_tot))
        return self.F, self.e_tot

    def algorithmic_bytes(self):
        p = self.plan
        s = 4 if p.dtype == ab.F32 else 8
        E, N, n, dV, dE = self.E, self.N, p.n, p.dV, p.dE
        feat, env = E * n * dV * s, N * n * dE * s
        return {"env_radial_forward": E * 3 * s + env, "tp_forward_energy": 2 * feat + env + E * s,
                "tp_backward_energy": (3 if self.gV is not None else 2) * feat + 2 * env,
                "tp_fused_energy": (2 if self.gV is not None else 1) * feat + 2 * env + E * s, "env_radial_backward": env + 2 * E * 3 * s,
                "force_gather": 2 * E * 3 * s + E * 4 + N * 3 * s, "segment_sum": E * s}


class TwoLayerStep:
    """One MD step of the stacked Allegro-style model of BASELINE.json:configs[2] (reading A19) as a sequence of library
    calls: edge embedding -> per layer [w = W_w x, env_embed, tensor product with dense per-path mix, latent update]
    -> readout of the l = 0 outputs -> the matching VJPs in reverse -> force gather.  `params` holds device tensors
    W_x0 [n,nb], W_v0 [n,nb], W_w [L,n,n], W_p [L,P,n,n], A_lat [L-1,n,2n], q [n] and floats rc, scale.
    `plan_last`: optional dense plan restricted to the 0e output block (Plan.set_out_blocks(1)) for the last layer, whose
    output feeds only the readout of the scalars: the paths into the other blocks are never run.
    `plan_first`: optional dense plan restricted to the natural-parity input blocks (Plan.set_in_blocks(0x19)) for the first
    layer, whose input V0 = v (x) Y has zeros in the other blocks (reading A19): half of the paths never run."""

    def __init__(self, plan_dense, plan_scalar, dev, params, plan_last=None, plan_first=None, sharded=None, fuse_readout=None, factorised_env=True):
        self.pd, self.ps, self.dev, self.p = plan_dense, plan_scalar, dev, params
        self.sharded = sharded      # sharding.ShardedForces: `dev` holds one rank's rows (see SingleLayerStep)
        # fuse_readout: the readout E = sum q . V_L[:, :, 0e] is taken in the last layer's forward epilogue and its cotangent formed inside
        # the last layer's VJP, so V_L is never stored (default: whenever the tcgen05 kernels serve the shape and plan_last is given)
        tc = plan_dense.dtype == ab.F32 and plan_dense.l_max == 2 and plan_dense.n == 64
        self.fuse_readout = (tc and plan_last is not None) if fuse_readout is None else (fuse_readout and tc)
        # layer-1 specialisation: V_0 = v0 (x) Y is generated on chip by the first layer's kernels (never stored), its cotangent arrives
        # contracted (g_v0, gY); needs the tensor-core kernels and a first-layer plan restricted to the natural-parity input blocks
        self.outer = tc and plan_first is not None and factorised_env and params["W_w"].shape[0] > 1
        self.factorised_env = factorised_env      # env-embed of the linear weights without forming w (False: linear + env_embed, the named calls)
        self.tc = tc      # tensor-core dense kernels: the 0e scalars travel between the layers in compact [E, n] side arrays
        self.pd_last = plan_last if plan_last is not None else plan_dense
        self.pd_first = plan_first if plan_first is not None else plan_dense
        self.L = params["W_w"].shape[0]
        rp, rvec = dev["row_ptr"], dev["rvec"]
        self.N, self.E = rp.shape[0] - 1, rvec.shape[0]
        dt, dv, n, dV = rvec.dtype, rvec.device, plan_dense.n, plan_dense.dV
        E, N, L = self.E, self.N, self.L
        new = lambda *shape: torch.empty(shape, dtype=dt, device=dv)
        self.x = [new(E, n) for _ in range(L)]            # x_0 .. x_{L-1}
        self.z = [new(E, n) for _ in range(L - 1)]
        self.V = [new(E, n, dV) for _ in range(L)] + [None if self.fuse_readout else new(E, n, dV)]    # V_0 .. V_L
        if self.outer:
            self.V[0] = None
            self.v0, self.g_v0, self.gY = new(E, n), new(E, n), new(E, plan_dense.dE)
        self.w = [new(E, n) for _ in range(L)]
        self.Eenv = [new(N, n, plan_dense.dE) for _ in range(L)]
        self.gEenv = new(N, n, plan_dense.dE)
        self.cot = [new(E, n, dV), new(E, n, dV)]          # ping-pong cotangents of V_l
        self.g_w, self.g_x, self.g_x2 = new(E, n), new(E, n), new(E, n)
        self.s = [new(E, n, 1) if self.tc else None for _ in range(L - 1)]      # compact V_{l+1}[:, :, 0e] for the latent update
        self.gs = new(E, n, 1) if (self.tc and L > 1) else None                  # compact cotangent of those scalars
        self.g_r, self.g_r_tmp = (new(E, 3) if sharded is None else sharded.g_local), new(E, 3)
        self.e_edge, self.e_tot, self.F = new(E), new(1), new(N, 3)
        self.e_ptr = torch.tensor([0, E], dtype=torch.int32, device=dv)
        self.ws = torch.empty(16, dtype=torch.uint8, device=dv)
        self.marks = None

    def run(self, mark=False):
        p, d, pd, ps, L = self.p, self.dev, self.pd, self.ps, self.L
        rp, rvec, rc, scale = d["row_ptr"], d["rvec"], p["rc"], p["scale"]
        ev = []

        def timed(name, fn):
            if not mark:
                return fn()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            r = fn()
            b.record()
            ev.append((name, a, b))
            return r

        if self.outer:
            timed("edge_embed", lambda: ab.edge_embed_factors(pd, rvec, p["W_x0"], p["W_v0"], rc, self.x[0], self.v0))
        else:
            timed("edge_embed", lambda: ab.edge_embed(pd, rvec, p["W_x0"], p["W_v0"], rc, x0=self.x[0], V0=self.V[0]))
        for l in range(L):
            if self.factorised_env:      # w = W_w x is never formed: the linear map is applied once per centre (allegro_env_linear_forward)
                timed("env_linear_forward", lambda: ab.env_linear_forward(ps, rp, rvec, self.x[l], p["W_w"][l], scale, Eenv=self.Eenv[l]))
            else:
                timed("linear", lambda: ab.linear(self.x[l], p["W_w"][l], y=self.w[l]))
                timed("env_embed", lambda: ab.env_embed(ps, rp, rvec, self.w[l], scale, Eenv=self.Eenv[l]))
            pl = self.pd_last if l == L - 1 else (self.pd_first if l == 0 else pd)
            if l == L - 1 and self.fuse_readout:
                timed("tp_forward_dense", lambda: ab.tp_forward_energy(pl, rp, self.V[l], self.Eenv[l], p["W_p"][l], p["q"], 0.0, want_out=False,
                                                                       want_G=False, e_edge=self.e_edge))
            elif self.outer and l == 0 and l < L - 1:
                timed("tp_forward_dense", lambda: ab.tp_forward_outer(pl, rp, rvec, self.v0, self.Eenv[l], p["W_p"][l], self.V[l + 1], self.s[l]))
            elif self.tc and l < L - 1:
                timed("tp_forward_dense", lambda: ab.tp_forward_aux(pl, rp, self.V[l], self.Eenv[l], p["W_p"][l], self.V[l + 1], self.s[l]))
            else:
                timed("tp_forward_dense", lambda: ab.tp_forward(pl, rp, self.V[l], self.Eenv[l], p["W_p"][l], out=self.V[l + 1]))
            if l < L - 1:
                Vs = self.s[l] if self.tc else self.V[l + 1]
                timed("latent_forward", lambda: ab.latent_forward(rvec, rc, self.x[l], Vs, p["A_lat"][l], z=self.z[l], x_new=self.x[l + 1]))
        # readout E = sum_e sum_n q[n] V_L[e][n][0e]; its cotangent q (x) delta_{k,0} is formed inside the last layer's VJP when
        # that kernel exists (fp32, l_max 2, n 64), otherwise materialised here
        fused_cot = pd.dtype == ab.F32 and pd.l_max == 2 and pd.n == 64
        G = self.V[L] if fused_cot else self.cot[0]
        if not self.fuse_readout:
            timed("edge_energy", lambda: ab.edge_energy(pd, self.V[L], p["q"], 0.0, e_edge=self.e_edge, want_G=not fused_cot, G=None if fused_cot else G))
        g_x_next, have_gr = None, False
        for l in reversed(range(L)):
            g_x = None
            if l < L - 1:     # x_{l+1} = u SiLU(A [x_l ; V_{l+1}[:,0e]]): cotangent g_x_next; adds to G[:, :, 0] and g_r
                g_x = self.g_x if g_x_next is not self.g_x else self.g_x2
                if self.tc:      # the scalars' cotangent goes into the compact side array; the dense VJP adds it to G while staging
                    self.gs.zero_()
                    timed("latent_backward", lambda: ab.latent_backward(rvec, rc, self.z[l], g_x_next, p["A_lat"][l], self.gs, self.g_r, g_x=g_x))
                else:
                    timed("latent_backward", lambda: ab.latent_backward(rvec, rc, self.z[l], g_x_next, p["A_lat"][l], G, self.g_r, g_x=g_x))
            gVl = self.cot[1] if G is self.cot[0] else self.cot[0]
            pl = self.pd_last if l == L - 1 else (self.pd_first if l == 0 else pd)
            if l == L - 1 and fused_cot:
                timed("tp_backward_dense", lambda: ab.tp_backward_energy(pl, rp, self.V[L], self.V[l], self.Eenv[l], p["W_p"][l], p["q"], 0.0, gV=gVl,
                                                                         gEenv=self.gEenv, workspace=self.ws))
            elif self.outer and l == 0 and l < L - 1:
                timed("tp_backward_dense", lambda: ab.tp_backward_outer(pl, rp, G, self.gs, rvec, self.v0, self.Eenv[l], p["W_p"][l], self.g_v0, self.gY,
                                                                        self.gEenv, workspace=self.ws))
            elif self.tc and l < L - 1:
                timed("tp_backward_dense", lambda: ab.tp_backward_aux(pl, rp, G, self.gs, self.V[l], self.Eenv[l], p["W_p"][l], gVl, self.gEenv,
                                                                      workspace=self.ws))
            else:
                timed("tp_backward_dense", lambda: ab.tp_backward(pl, rp, G, self.V[l], self.Eenv[l], p["W_p"][l], gV=gVl, gEenv=self.gEenv, workspace=self.ws))
            if self.factorised_env:
                acc_x = g_x is not None
                if g_x is None:
                    g_x = self.g_x if g_x_next is not self.g_x else self.g_x2
                timed("env_linear_backward", lambda: ab.env_linear_backward(ps, rp, self.gEenv, rvec, self.x[l], p["W_w"][l], scale, self.g_r, g_x,
                                                                            accumulate_g_rvec=have_gr, accumulate_g_x=acc_x))
                have_gr = True
            else:
                if not have_gr:
                    timed("env_embed_backward", lambda: ab.env_embed_backward(ps, rp, self.gEenv, rvec, self.w[l], scale, g_rvec=self.g_r, g_w=self.g_w))
                    have_gr = True
                else:
                    timed("env_embed_backward", lambda: ab.env_embed_backward(ps, rp, self.gEenv, rvec, self.w[l], scale, g_rvec=self.g_r_tmp, g_w=self.g_w))
                    timed("add_inplace", lambda: ab.add_inplace(self.g_r, self.g_r_tmp))
                if g_x is None:
                    g_x = self.g_x if g_x_next is not self.g_x else self.g_x2
                    timed("linear", lambda: ab.linear(self.g_w, p["W_w"][l], transpose_w=True, y=g_x))
                else:
                    timed("linear", lambda: ab.linear(self.g_w, p["W_w"][l], transpose_w=True, y=g_x, accumulate=True))
            G, g_x_next = gVl, g_x
        if self.outer and L > 1:
            timed("edge_embed_backward", lambda: ab.edge_embed_factors_backward(pd, rvec, p["W_x0"], p["W_v0"], rc, g_x_next, self.g_v0, self.gY, self.g_r))
        else:
            timed("edge_embed_backward", lambda: ab.edge_embed_backward(pd, rvec, p["W_x0"], p["W_v0"], rc, g_x_next, G, self.g_r))
        if self.sharded is None:
            timed("force_gather", lambda: ab.force_gather(rp, d["rev"], self.g_r, F=self.F))
            timed("segment_sum", lambda: ab.segment_sum(self.e_ptr, self.e_edge, out=self.e_tot))
        else:
            timed("halo_exchange", self.sharded.exchange)
            timed("force_gather", lambda: ab.force_gather(rp, d["rev"], self.sharded.g_ext, F=self.F))
            timed("segment_sum", lambda: ab.segment_sum(self.e_ptr, self.e_edge, out=self.e_tot))
            timed("energy_all_reduce", lambda: self.sharded.reduce_sum(self.e_tot))
        self.marks = ev
        return self.F, self.e_tot

    def algorithmic_bytes(self):
        """HBM bytes the dense tensor-product calls must move at least once (V in, out out; VJP: cotangent and V in,
        gV out; Eenv / gEenv per centre), summed over layers"""
        pd = self.pd
        s = 4 if pd.dtype == ab.F32 else 8
        feat, env = self.E * pd.n * pd.dV * s, self.N * pd.n * pd.dE * s
        return {"tp_forward_dense": self.L * (2 * feat + env), "tp_backward_dense": self.L * (3 * feat + 2 * env)}

    def algorithmic_flops(self):
        """FP32 flops the dense tensor-product calls must execute (sparse CG 806 flop per channel-edge forward,
        twice that for the VJP; per-path n x n mix 2 n^2 sum_p (2 l3 + 1) per edge), per call name, summed over layers"""
        pd = self.pd
        n, L = pd.n, self.L
        cg_fwd = {1: 2 * 32 + 32, 2: 2 * 274 + 258, 3: 2 * 1222 + 1082}[pd.l_max] * n
        dT = {1: 22, 2: 102, 3: 312}[pd.l_max]
        mix = 2 * n * n * dT
        return {"tp_forward_dense": L * self.E * (cg_fwd + mix), "tp_backward_dense": L * self.E * (2 * cg_fwd + mix)}


def shard_to_device(inp, sharded, keys_edge=("rvec", "V"), keys_full=("W_r", "path_w", "q"), device="cuda"):
    """One rank's rows of the host problem `inp` as device tensors: row_ptr / rev become the rank-local index arrays of the
    HaloPlan, per-edge tensors are sliced to the rank's edge range [e0, e1), parameters are replicated."""
    hp = sharded.plan
    dev = dict(row_ptr=torch.from_numpy(hp.row_ptr_loc).to(device), rev=torch.from_numpy(hp.rev_loc).to(device))
    for k in keys_edge:
        if inp.get(k) is not None:
            v = inp[k][hp.e0:hp.e1]
            dev[k] = (v if hasattr(v, "detach") else torch.from_numpy(np.ascontiguousarray(v))).to(device).contiguous()
    for k in keys_full:
        if inp.get(k) is not None:
            v = inp[k]
            dev[k] = (v if hasattr(v, "detach") else torch.from_numpy(np.ascontiguousarray(v))).to(device)
    return dev


class GraphedStep:
    """A step object (SingleLayerStep / TwoLayerStep / ChunkedStep) captured once into a CUDA graph and replayed: one graph
    launch per MD step instead of 8-30 kernel launches, which is what bounds small systems (the paper's 25-100 atom
    molecules).  Buffers are the wrapped step's own (allocated once), so replays read the current contents
    of dev["rvec"], dev["V"], ... and overwrite F / e_tot in place."""

    def __init__(self, step, warmup=3):
        self.step = step
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):       # warm up on the capture stream (first calls set function attributes)
            for _ in range(warmup):
                step.run()
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        self.graph = torch.cuda.CUDAGraph()
        n0 = ab.launch_count()
        with torch.cuda.graph(self.graph):
            step.run()
        self.kernels_per_step = ab.launch_count() - n0      # kernel nodes of the graph = kernels each replay launches
        self.F, self.e_tot = step.F, step.e_tot
        self.marks = None

    def run(self, mark=False):
        self.graph.replay()
        return self.F, self.e_tot

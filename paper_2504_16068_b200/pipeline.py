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

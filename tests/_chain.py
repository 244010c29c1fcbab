"""Shared by the parity tests, smoke() and bench.py: the single-layer chain of the scalar-weight configs
(C0, C1, C3, C4 and their reduced variants) evaluated (a) by the float64 oracle and (b) by the CUDA
library, on the same seeded inputs.

Chain (reading A12 for the energy):
    w = radial(r)  ->  Eenv = env_embed(w)  ->  out = tp_forward(V, Eenv, path_w)
    -> e_edge, G = edge_energy(out, q, kappa)  ->  gV, gEenv, g_path_w = tp_backward(G, ...)
    -> g_r, g_w = env_embed_backward(gEenv)  ->  g_r += radial_backward(g_w)  ->  F = force_gather(g_r)
    (C4: E_mol = segment_sum over the edges of each molecule's centres)

Inputs are generated in float64, rounded ONCE to the config's dtype; the oracle consumes the rounded
values promoted to double (reading A9), so differences isolate the kernels' arithmetic.
No arithmetic of the method lives here: only calls into oracle/ (CPU side) or the library (GPU side).
"""
import numpy as np

from paper_2504_16068_b200.pipeline import gpu_chain, to_device  # noqa: F401
from workloads.inputs import make_inputs, sub_inputs  # noqa: F401


def oracle_chain(inp, centres=None, want_gw=True, forces=True):
    """float64 reference.  With centres=(c_lo, c_hi) the per-edge / per-centre tensors are computed for those
    centres only (rows outside are zero) and F / E_mol are omitted."""
    import oracle as orc
    f8 = lambda a: np.asarray(a, dtype=np.float64)
    lmax, rp = inp["lmax"], inp["row_ptr"]
    rvec, V, pw, q = f8(inp["rvec"]), f8(inp["V"]), f8(inp["path_w"]), f8(inp["q"])
    w, dwdr = orc.radial(f8(inp["W_r"]), inp["rc"], rvec)
    Eenv = orc.env_embed(lmax, rp, rvec, w, inp["scale"])
    out = orc.tp_forward(lmax, rp, V, Eenv, pw, centres=centres)
    e_edge, G = orc.edge_energy(lmax, out, q, inp["kappa"])
    gV, gE, gpw = orc.tp_backward(lmax, rp, G, V, Eenv, pw, want_gV=True, want_gw=want_gw, centres=centres)
    g_r, g_w = orc.env_embed_backward(lmax, rp, gE, rvec, w, inp["scale"], centres=centres)
    g_r_env = g_r.copy()
    orc.radial_backward(rvec, g_w, dwdr, g_r)
    res = dict(w=w, Eenv=Eenv, out=out, e_edge=e_edge, G=G, gV=gV, gEenv=gE, g_path_w=gpw, g_w=g_w, g_r_env=g_r_env, g_r=g_r)
    if centres is None and forces:
        res["F"] = orc.force_gather(rp, inp["rev"], g_r)
        if inp.get("edge_mol_ptr") is not None:
            res["E_mol"] = orc.segment_sum(inp["edge_mol_ptr"], e_edge)
    return res


# tolerances of BASELINE.json:north_star (reading A10): per tensor max|d| <= tol * max|ref|
TOL = {np.float32: 1e-5, np.float64: 1e-11}
FORCE_RMS_TOL = {np.float32: 1e-4, np.float64: 1e-10}


def compare(ref, got, dt, keys=None, rows=None):
    """-> {key: max|d| / max|ref|}; `rows` (slice) restricts per-edge tensors, given as dict key -> slice."""
    errs = {}
    for k in (keys or ref.keys()):
        if k not in got or got[k] is None or ref.get(k) is None:
            continue
        r = np.asarray(ref[k], dtype=np.float64)
        g = got[k]
        g = g.detach().cpu().numpy().astype(np.float64) if hasattr(g, "detach") else np.asarray(g, dtype=np.float64)
        if rows is not None and k in rows:
            r, g = r[rows[k]], g[rows[k]]
        den = np.max(np.abs(r)) if r.size else 1.0
        errs[k] = float(np.max(np.abs(r - g)) / den) if r.size and den > 0 else 0.0
    return errs

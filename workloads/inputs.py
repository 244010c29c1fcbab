"""Seeded inputs of the single-layer chain of the scalar-weight configs (C0, C1, C3, C4 and reduced variants).

Generated in float64 and rounded ONCE to the config's dtype; both the oracle (which promotes them back to
double, reading A9) and the CUDA library consume these arrays.  No arithmetic of the method lives here.

features="host"   : V is a numpy array (small configs).
features="lazy"   : V is not materialised; sub_inputs() draws the rows it needs (CPU-only timing of a sample).
features="device" : V is drawn directly in device memory by the torch form of the same counter-based
                    generator (full-size configs: C1 is 1.7 GB, C3 86 GB per tensor); whoever needs exact
                    values on the host (the oracle, for the centres it checks) reads them back with
                    sub_inputs(), so both sides consume identical bits.
"""
import numpy as np

from . import configs, rng


def make_inputs(name, seed=0, features="host", device="cuda"):
    g = configs.geometry_for(name, seed)
    s = g["spec"]
    wts = configs.weights_for(name, seed)
    dt = configs.np_dtype(name)
    E = g["rvec"].shape[0]
    inp = dict(name=name, spec=s, dt=dt, lmax=s["lmax"], n=s["n"], rc=s["rc"], N=g["row_ptr"].shape[0] - 1, E=E,
               row_ptr=g["row_ptr"], rev=g["rev"], mol_ptr=g["mol_ptr"],
               rvec=np.ascontiguousarray(g["rvec"].astype(dt)),
               W_r=np.ascontiguousarray(wts["W_r"].astype(dt)),
               path_w=np.ascontiguousarray(wts["path_w"].astype(dt)),
               q=np.ascontiguousarray(wts["q"].astype(dt)), kappa=wts["kappa"], scale=1.0)
    inp["seed"] = seed
    if features == "host":
        inp["V"] = np.ascontiguousarray(configs.features_for(name, E, seed, "V").astype(dt))
    elif features == "lazy":      # rows are drawn on demand by sub_inputs() (a pure function of the edge index)
        inp["V"] = None
    else:
        import torch
        dV = 2 * (s["lmax"] + 1) ** 2
        inp["V"] = rng.normal_torch(seed, rng.STREAMS["V"], (E, s["n"], dV), device=device,
                                    dtype=torch.float32 if dt == np.float32 else torch.float64)
    if g["mol_ptr"] is not None:
        inp["edge_mol_ptr"] = g["row_ptr"][g["mol_ptr"]].astype(np.int32)
    return inp


def sub_inputs(inp, c_lo, c_hi):
    """The self-contained sub-problem of centres [c_lo, c_hi) with their complete neighbourhoods (host arrays).
    Every per-edge and per-centre quantity of the chain depends on one centre only (strict locality), so the
    sub-problem's results equal rows [row_ptr[c_lo], row_ptr[c_hi]) / [c_lo, c_hi) of the full problem's.
    Forces are not defined on a sub-problem (reverse edges belong to other centres)."""
    rp = inp["row_ptr"]
    e0, e1 = int(rp[c_lo]), int(rp[c_hi])
    if inp["V"] is None:
        V = configs.features_for(inp["name"], inp["E"], inp["seed"], "V", e0, e1).astype(inp["dt"])
    else:
        V = inp["V"][e0:e1]
    if hasattr(V, "detach"):
        V = V.detach().cpu().numpy()
    sub = dict(inp)
    sub.update(N=c_hi - c_lo, E=e1 - e0, row_ptr=(rp[c_lo:c_hi + 1] - rp[c_lo]).astype(np.int32), rev=None, mol_ptr=None,
               rvec=np.ascontiguousarray(inp["rvec"][e0:e1]), V=np.ascontiguousarray(V), edge_range=(e0, e1),
               centre_range=(c_lo, c_hi))
    sub.pop("edge_mol_ptr", None)
    return sub


def make_model_inputs(name, seed=0, n=None, lmax=None, n_layers=None):
    """Inputs of the two-layer model of configs[2] (reading A19): geometry of config `name` plus the dense weights.
    n / lmax / n_layers override the config's (small oracle-only pins).  Weights are float64 here; each side rounds
    them to its dtype.  scale = 1/sqrt(E/N) (reading A6)."""
    g = configs.geometry_for(name, seed)
    s = dict(g["spec"])
    n = n or s["n"]
    lmax = lmax or s["lmax"]
    L = n_layers or s.get("n_layers", 2)
    P = configs.num_paths(lmax)
    S = rng.STREAMS
    nb = configs.N_BASIS
    E, N = g["rvec"].shape[0], g["row_ptr"].shape[0] - 1
    dt = configs.np_dtype(name)
    params = dict(
        lmax=lmax, n=n, nb=nb, n_layers=L, rc=s["rc"], scale=1.0 / np.sqrt(E / N),
        W_x0=rng.normal(seed, S["W_x0"], (n, nb)) / np.sqrt(nb),
        W_v0=rng.normal(seed, S["W_v0"], (n, nb)) / np.sqrt(nb),
        W_w=rng.normal(seed, S["W_w"], (L, n, n)) / np.sqrt(n),
        W_p=rng.normal(seed, S["W_p"], (L, P, n, n)) / np.sqrt(n),
        A_lat=rng.normal(seed, S["A_lat"], (max(L - 1, 1), n, 2 * n)) / np.sqrt(2 * n),
        q=rng.normal(seed, S["q"], (n,)) / np.sqrt(n),
    )
    for k in ("W_x0", "W_v0", "W_w", "W_p", "A_lat", "q"):      # rounded once to the config's dtype (reading A9)
        params[k] = np.ascontiguousarray(params[k].astype(dt)).astype(np.float64) if dt == np.float32 else params[k]
    return dict(name=name, dt=dt, N=N, E=E, row_ptr=g["row_ptr"], rev=g["rev"], rvec=np.ascontiguousarray(g["rvec"].astype(dt)),
                params=params)

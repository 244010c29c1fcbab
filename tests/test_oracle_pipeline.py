"""Pins for the oracle's pipeline (env-embed, tensor product, VJPs, forces): brute force on
tiny inputs, equivariance under proper and improper rotations via Wigner-D, parity selection,
path isolation, adjoint identities, central finite differences of the energy, sum F = 0,
segment plan by brute force.  CPU only; the CUDA path is not involved.
"""
import numpy as np
import pytest

import oracle
from workloads import configs, rng


def _small_graph(name="C0", n=None, lmax=None, seed=0):
    g = configs.geometry_for(name, seed)
    s = dict(g["spec"])
    if n is not None:
        s["n"] = n
    if lmax is not None:
        s["lmax"] = lmax
    g["spec"] = s
    return g


def _rand_inputs(g, seed=0, dense=False):
    s = g["spec"]
    n, lmax = s["n"], s["lmax"]
    E = g["rvec"].shape[0]
    dV = 2 * (lmax + 1) ** 2
    P = configs.num_paths(lmax)
    rs = np.random.RandomState(seed + 11)
    V = rs.randn(E, n, dV)
    G = rs.randn(E, n, dV)
    Wr = rs.randn(n, 8) / np.sqrt(8)
    pw = rs.randn(P, n, n) / np.sqrt(n) if dense else rs.randn(P) / np.sqrt(P)
    q = rs.randn(n) / np.sqrt(n)
    return V, G, Wr, pw, q


def _blockdiag_D(lmax, a, b, c, improper=False):
    """feature-space rotation: D^l on every (l, parity) block; inversion multiplies odd blocks by -1"""
    dV = 2 * (lmax + 1) ** 2
    M = np.zeros((dV, dV))
    for l in range(lmax + 1):
        D = oracle.wigner_D_real(l, a, b, c)
        for p in (0, 1):
            off = 2 * l * l + (2 * l + 1 if p else 0)
            sgn = -1.0 if (improper and p == 1) else 1.0
            M[off:off + 2 * l + 1, off:off + 2 * l + 1] = sgn * D
    return M


def _env_D(lmax, a, b, c, improper=False):
    dE = (lmax + 1) ** 2
    M = np.zeros((dE, dE))
    for l in range(lmax + 1):
        sgn = (-1.0) ** l if improper else 1.0
        M[l * l:(l + 1) ** 2, l * l:(l + 1) ** 2] = sgn * oracle.wigner_D_real(l, a, b, c)
    return M


# ----------------------------------------------------------------------------- forward

@pytest.mark.parametrize("lmax,n", [(1, 3), (2, 2), (3, 2)])
def test_tp_forward_brute_force_numpy(lmax, n):
    """dense oracle == sparse oracle == an einsum over the (separately pinned) real-CG blocks"""
    g = _small_graph("C0", n=n, lmax=lmax)
    V, G, Wr, pw, q = _rand_inputs(g)
    w, _ = oracle.radial(Wr, g["spec"]["rc"], g["rvec"])
    Eenv = oracle.env_embed(lmax, g["row_ptr"], g["rvec"], w, 0.7)
    # env-embed by brute force
    Y = np.array([oracle.sph_harm(lmax, r)[0] for r in g["rvec"]])
    Eb = np.zeros_like(Eenv)
    for e, c in enumerate(g["centre"]):
        Eb[c] += 0.7 * w[e][:, None] * Y[e][None, :]
    assert np.allclose(Eenv, Eb, atol=1e-13)
    out_d = oracle.tp_forward(lmax, g["row_ptr"], V, Eenv, pw, variant="dense")
    out_s = oracle.tp_forward(lmax, g["row_ptr"], V, Eenv, pw, variant="sparse")
    p = oracle.paths(lmax)
    ref = np.zeros_like(V)
    Ee = Eenv[g["centre"]]
    for t in range(len(pw)):
        l1, l2, l3 = int(p["l1"][t]), int(p["l2"][t]), int(p["l3"][t])
        C, _, _ = oracle.cg_real(l1, l2, l3)
        o1, o2, o3 = int(p["off1"][t]), int(p["off2"][t]), int(p["off3"][t])
        ref[:, :, o3:o3 + 2 * l3 + 1] += pw[t] * np.einsum("abM,ena,enb->enM", C, V[:, :, o1:o1 + 2 * l1 + 1],
                                                           Ee[:, :, o2:o2 + 2 * l2 + 1])
    assert np.allclose(out_d, ref, atol=1e-12)
    assert np.allclose(out_s, ref, atol=1e-12)


def test_tp_dense_mode_brute_force_and_reduction_to_scalar():
    lmax, n = 2, 3
    g = _small_graph("C0", n=n, lmax=lmax)
    V, G, Wr, pwd, q = _rand_inputs(g, dense=True)
    _, _, _, pws, _ = _rand_inputs(g, dense=False)
    w, _ = oracle.radial(Wr, g["spec"]["rc"], g["rvec"])
    Eenv = oracle.env_embed(lmax, g["row_ptr"], g["rvec"], w)
    # W[p] = w_p I reproduces scalar mode
    Wd = pws[:, None, None] * np.eye(n)[None]
    a = oracle.tp_forward(lmax, g["row_ptr"], V, Eenv, Wd, variant="sparse")
    b = oracle.tp_forward(lmax, g["row_ptr"], V, Eenv, pws, variant="sparse")
    assert np.allclose(a, b, atol=1e-13)
    # general W by einsum
    p = oracle.paths(lmax)
    ref = np.zeros_like(V)
    Ee = Eenv[g["centre"]]
    for t in range(pwd.shape[0]):
        l1, l2, l3 = int(p["l1"][t]), int(p["l2"][t]), int(p["l3"][t])
        C, _, _ = oracle.cg_real(l1, l2, l3)
        o1, o2, o3 = int(p["off1"][t]), int(p["off2"][t]), int(p["off3"][t])
        tt = np.einsum("abM,ena,enb->enM", C, V[:, :, o1:o1 + 2 * l1 + 1], Ee[:, :, o2:o2 + 2 * l2 + 1])
        ref[:, :, o3:o3 + 2 * l3 + 1] += np.einsum("on,enM->eoM", pwd[t], tt)
    for variant in ("dense", "sparse"):
        assert np.allclose(oracle.tp_forward(lmax, g["row_ptr"], V, Eenv, pwd, variant=variant), ref, atol=1e-12)


@pytest.mark.parametrize("lmax", [1, 2, 3])
@pytest.mark.parametrize("improper", [False, True])
def test_equivariance_wigner_D(lmax, improper):
    """out(D V, env(R r)) = D out to 1e-12 (north_star), for rotations and rotation x inversion"""
    n = 2
    g = _small_graph("C0", n=n, lmax=lmax)
    V, G, Wr, pw, q = _rand_inputs(g)
    a, b, c = 0.81, 1.37, -2.2
    R = oracle.rotation_matrix(a, b, c) * (-1.0 if improper else 1.0)
    DV = _blockdiag_D(lmax, a, b, c, improper)
    DE = _env_D(lmax, a, b, c, improper)
    w, _ = oracle.radial(Wr, g["spec"]["rc"], g["rvec"])
    E0 = oracle.env_embed(lmax, g["row_ptr"], g["rvec"], w)
    rv1 = g["rvec"] @ R.T
    w1, _ = oracle.radial(Wr, g["spec"]["rc"], rv1)
    assert np.allclose(w, w1, atol=1e-13)
    E1 = oracle.env_embed(lmax, g["row_ptr"], rv1, w1)
    assert np.allclose(E1, E0 @ DE.T, atol=1e-12)
    out0 = oracle.tp_forward(lmax, g["row_ptr"], V, E0, pw)
    out1 = oracle.tp_forward(lmax, g["row_ptr"], V @ DV.T, E1, pw)
    assert np.abs(out1 - out0 @ DV.T).max() < 1e-12 * max(1.0, np.abs(out0).max())
    # invariant energy when V transforms as a tensor
    e0, _ = oracle.edge_energy(lmax, out0, q, 0.3)
    e1, _ = oracle.edge_energy(lmax, out1, q, 0.3)
    assert np.allclose(e0, e1, atol=1e-11)


def test_path_isolation_and_parity_selection():
    lmax, n = 2, 2
    g = _small_graph("C0", n=n, lmax=lmax)
    V, G, Wr, pw, q = _rand_inputs(g)
    w, _ = oracle.radial(Wr, g["spec"]["rc"], g["rvec"])
    Eenv = oracle.env_embed(lmax, g["row_ptr"], g["rvec"], w)
    p = oracle.paths(lmax)
    total = np.zeros_like(V)
    for t in range(len(pw)):
        one = np.zeros_like(pw)
        one[t] = pw[t]
        o = oracle.tp_forward(lmax, g["row_ptr"], V, Eenv, one)
        l3, o3 = int(p["l3"][t]), int(p["off3"][t])
        mask = np.ones(V.shape[2], bool)
        mask[o3:o3 + 2 * l3 + 1] = False
        assert np.abs(o[:, :, mask]).max() == 0.0          # only the path's own output block is touched
        # and only its own input block matters
        V2 = V.copy()
        l1, o1 = int(p["l1"][t]), int(p["off1"][t])
        keep = np.zeros(V.shape[2], bool)
        keep[o1:o1 + 2 * l1 + 1] = True
        V2[:, :, ~keep] = 0.0
        assert np.array_equal(oracle.tp_forward(lmax, g["row_ptr"], V2, Eenv, one), o)
        total += o
    assert np.allclose(total, oracle.tp_forward(lmax, g["row_ptr"], V, Eenv, pw), atol=1e-13)
    assert np.abs(oracle.tp_forward(lmax, g["row_ptr"], V, Eenv, np.zeros_like(pw))).max() == 0.0


# ----------------------------------------------------------------------------- VJP

@pytest.mark.parametrize("dense", [False, True])
def test_tp_backward_adjoint_identities(dense):
    lmax, n = 2, 3
    g = _small_graph("C0", n=n, lmax=lmax)
    V, G, Wr, pw, q = _rand_inputs(g, dense=dense)
    w, _ = oracle.radial(Wr, g["spec"]["rc"], g["rvec"])
    Eenv = oracle.env_embed(lmax, g["row_ptr"], g["rvec"], w)
    gV, gE, gw = oracle.tp_backward(lmax, g["row_ptr"], G, V, Eenv, pw)
    rs = np.random.RandomState(5)
    dVv, dEe, dw = rs.randn(*V.shape), rs.randn(*Eenv.shape), rs.randn(*pw.shape)
    fw = lambda V_, E_, w_: oracle.tp_forward(lmax, g["row_ptr"], V_, E_, w_)
    # the product is linear in each of V, Eenv, path_w separately
    assert abs((G * fw(dVv, Eenv, pw)).sum() - (gV * dVv).sum()) < 1e-9
    assert abs((G * fw(V, dEe, pw)).sum() - (gE * dEe).sum()) < 1e-9
    assert abs((G * fw(V, Eenv, dw)).sum() - (gw * dw).sum()) < 1e-9
    # gV = None path gives the same gE
    _, gE2, _ = oracle.tp_backward(lmax, g["row_ptr"], G, V, Eenv, pw, want_gV=False, want_gw=False)
    assert np.array_equal(gE, gE2)
    # centre sub-range touches only its own rows and equals the full result there
    gV3, gE3, _ = oracle.tp_backward(lmax, g["row_ptr"], G, V, Eenv, pw, centres=(5, 9), want_gw=False)
    e0, e1 = g["row_ptr"][5], g["row_ptr"][9]
    assert np.array_equal(gV3[e0:e1], gV[e0:e1]) and np.abs(gV3[:e0]).max() == 0 and np.abs(gV3[e1:]).max() == 0
    assert np.array_equal(gE3[5:9], gE[5:9]) and np.abs(gE3[:5]).max() == 0


def test_env_embed_backward_adjoint_and_fd():
    lmax, n = 3, 2
    g = _small_graph("C0", n=n, lmax=lmax)
    rs = np.random.RandomState(7)
    E = g["rvec"].shape[0]
    w = rs.randn(E, n)
    gE = rs.randn(len(g["row_ptr"]) - 1, n, (lmax + 1) ** 2)
    g_r, g_w = oracle.env_embed_backward(lmax, g["row_ptr"], gE, g["rvec"], w, 0.9)
    dw = rs.randn(E, n)
    lin = oracle.env_embed(lmax, g["row_ptr"], g["rvec"], dw, 0.9)
    assert abs((gE * lin).sum() - (g_w * dw).sum()) < 1e-10
    f = lambda rv: (gE * oracle.env_embed(lmax, g["row_ptr"], rv, w, 0.9)).sum()
    for e in (0, 17, E - 1):
        for a in range(3):
            h = 1e-6
            rp, rm = g["rvec"].copy(), g["rvec"].copy()
            rp[e, a] += h
            rm[e, a] -= h
            assert abs((f(rp) - f(rm)) / (2 * h) - g_r[e, a]) < 2e-7 * max(1.0, abs(g_r[e, a]))


def _energy_and_forces(g, pos, V, Wr, pw, q, kappa, shift, scale=1.0):
    s = g["spec"]
    lmax = s["lmax"]
    rvec = pos[g["col"]] - pos[g["centre"]] + shift
    w, dw = oracle.radial(Wr, s["rc"], rvec)
    Eenv = oracle.env_embed(lmax, g["row_ptr"], rvec, w, scale)
    out = oracle.tp_forward(lmax, g["row_ptr"], V, Eenv, pw)
    e_edge, G = oracle.edge_energy(lmax, out, q, kappa)
    etot = e_edge.sum()
    _, gE, _ = oracle.tp_backward(lmax, g["row_ptr"], G, V, Eenv, pw, want_gV=False, want_gw=False)
    g_r, g_w = oracle.env_embed_backward(lmax, g["row_ptr"], gE, rvec, w, scale)
    oracle.radial_backward(rvec, g_w, dw, g_r)
    F = oracle.force_gather(g["row_ptr"], g["rev"], g_r)
    return etot, F


@pytest.mark.parametrize("name,lmax,n,dense", [("C0", 1, 8, False), ("C0", 2, 3, False), ("C0", 3, 2, False),
                                              ("C0", 2, 3, True), ("C4s", 2, 2, False)])
def test_forces_vs_central_differences(name, lmax, n, dense):
    """F = -dE_tot/dx through radial, env-embed and the tensor product; sum F = 0 (north_star)."""
    g = _small_graph(name, n=n, lmax=lmax)
    V, G, Wr, pw, q = _rand_inputs(g, dense=dense)
    pos = g["pos"].copy()
    shift = g["rvec"] - (pos[g["col"]] - pos[g["centre"]])
    e0, F = _energy_and_forces(g, pos, V, Wr, pw, q, 0.3, shift)
    assert np.abs(F.sum(0)).max() < 1e-11 * max(1.0, np.abs(F).max())
    h = 1e-5
    rs = np.random.RandomState(3)
    for a in rs.choice(pos.shape[0], 4, replace=False):
        for d in range(3):
            pp, pm = pos.copy(), pos.copy()
            pp[a, d] += h
            pm[a, d] -= h
            ep, _ = _energy_and_forces(g, pp, V, Wr, pw, q, 0.3, shift)
            em, _ = _energy_and_forces(g, pm, V, Wr, pw, q, 0.3, shift)
            fd = -(ep - em) / (2 * h)
            assert abs(fd - F[a, d]) < 5e-7 * max(1.0, np.abs(F).max()), (a, d, fd, F[a, d])


def test_path_weight_gradient_vs_fd():
    lmax, n = 2, 2
    g = _small_graph("C4s", n=n, lmax=lmax)
    V, G, Wr, pw, q = _rand_inputs(g)
    w, _ = oracle.radial(Wr, g["spec"]["rc"], g["rvec"])
    Eenv = oracle.env_embed(lmax, g["row_ptr"], g["rvec"], w)

    def en(pw_):
        out = oracle.tp_forward(lmax, g["row_ptr"], V, Eenv, pw_)
        e, G_ = oracle.edge_energy(lmax, out, q, 0.3)
        return e.sum(), G_
    e0, G0 = en(pw)
    _, _, gw = oracle.tp_backward(lmax, g["row_ptr"], G0, V, Eenv, pw, want_gV=False)
    for t in (0, 7, 29):
        h = 1e-6
        a, b = pw.copy(), pw.copy()
        a[t] += h
        b[t] -= h
        fd = (en(a)[0] - en(b)[0]) / (2 * h)
        assert abs(fd - gw[t]) < 1e-6 * max(1.0, abs(gw[t]))
    # per-molecule energies: segment sums over atoms == brute force over edges
    e_edge, _ = oracle.edge_energy(lmax, oracle.tp_forward(lmax, g["row_ptr"], V, Eenv, pw), q, 0.3)
    e_atom = oracle.segment_sum(g["row_ptr"], e_edge)
    e_mol = oracle.segment_sum(g["mol_ptr"], e_atom)
    mol_of_atom = np.searchsorted(g["mol_ptr"], np.arange(len(e_atom)), side="right") - 1
    ref = np.zeros(len(g["mol_ptr"]) - 1)
    np.add.at(ref, mol_of_atom[g["centre"]], e_edge)
    assert np.allclose(e_mol, ref, atol=1e-10) and abs(e_mol.sum() - e0) < 1e-9


def test_edge_energy_cotangent():
    rs = np.random.RandomState(9)
    out = rs.randn(7, 3, 18)
    q = rs.randn(3)
    e, G = oracle.edge_energy(2, out, q, 0.3)
    ref = (q[None, :] * out[:, :, 0]).sum(1) + 0.15 * (out ** 2).sum((1, 2))
    assert np.allclose(e, ref, atol=1e-13)
    Gref = 0.3 * out
    Gref[:, :, 0] += q[None, :]
    assert np.allclose(G, Gref, atol=1e-15)


# ----------------------------------------------------------------------------- integers

def test_segment_plan_brute_force():
    rs = np.random.RandomState(10)
    deg = rs.randint(0, 40, size=50)
    deg[[3, 10]] = 0
    deg[7] = 300
    row_ptr = np.concatenate([[0], np.cumsum(deg)]).astype(np.int32)
    for T in (1, 8, 32, 128):
        items = oracle.segments(row_ptr, T)
        ref = []
        for i, d in enumerate(deg):
            if d == 0:
                ref.append((i, row_ptr[i], row_ptr[i]))
            for k in range(-(-d // T)):
                e0 = row_ptr[i] + k * T
                ref.append((i, e0, min(e0 + T, row_ptr[i + 1])))
        assert items.tolist() == [list(map(int, r)) for r in ref]
        covered = np.concatenate([np.arange(a, b) for _, a, b in items] + [np.zeros(0, int)])
        assert np.array_equal(covered, np.arange(row_ptr[-1]))


def test_generated_neighbour_lists_are_valid():
    for name in ("C0", "C4s"):
        g = configs.geometry_for(name)
        rp, col, ctr, rev, rv = g["row_ptr"], g["col"], g["centre"], g["rev"], g["rvec"]
        r = np.linalg.norm(rv, axis=1)
        assert (r > 0).all() and (r < g["spec"]["rc"]).all()
        assert np.array_equal(col[rev], ctr) and np.array_equal(ctr[rev], col)
        assert np.abs(rv + rv[rev]).max() == 0.0
        for i in range(len(rp) - 1):
            assert np.all(np.diff(col[rp[i]:rp[i + 1]]) > 0)
        # brute-force pair search
        pos = g["pos"]
        d = pos[None] - pos[:, None]
        if g["box"]:
            d -= g["box"] * np.round(d / g["box"])
        dist = np.sqrt((d ** 2).sum(-1))
        adj = (dist < g["spec"]["rc"]) & (dist > 0)
        if g["mol_ptr"] is not None:
            mol = np.searchsorted(g["mol_ptr"], np.arange(len(pos)), side="right") - 1
            adj &= mol[:, None] == mol[None, :]
        ii, jj = np.nonzero(adj)
        assert np.array_equal(ii, ctr) and np.array_equal(jj, col)
        assert np.allclose(d[ii, jj], rv, atol=1e-12)


def test_virial_is_the_strain_derivative_of_the_energy():
    """orc.virial (reading A25) pinned by central finite differences: deform every edge vector by r -> (I + h e_a e_b^T) r, re-evaluate
    the whole chain's energy (radial weights, embedding, tensor product, energy) and difference; all nine components, plus the
    closed form trace(W) = sum_e r_e . g_r[e] = dE/d(ln scale).  The configs' boxes play no role: the energy sees positions only
    through the edge vectors."""
    import _chain
    inp = _chain.make_inputs("C0")
    base = _chain.oracle_chain(inp, want_gw=False)
    W = oracle.virial(inp["rvec"].astype(np.float64), base["g_r"])
    assert W.shape == (3, 3)
    assert abs(np.trace(W) - float(np.sum(inp["rvec"].astype(np.float64) * base["g_r"]))) <= 1e-12 * abs(np.trace(W))

    def energy(defo):
        sub = dict(inp)
        sub["rvec"] = inp["rvec"].astype(np.float64) @ defo.T
        return float(np.sum(_chain.oracle_chain(sub, want_gw=False, forces=False)["e_edge"]))

    h = 1e-6
    for a in range(3):
        for b in range(3):
            d = np.zeros((3, 3))
            d[a, b] = h
            fd = (energy(np.eye(3) + d) - energy(np.eye(3) - d)) / (2 * h)
            assert abs(fd - W[a, b]) <= 2e-7 * np.abs(W).max(), (a, b, fd, W[a, b])
    # W is NOT symmetric here (V ~ N(0,1) does not rotate with the geometry, so E_tot is not rotation invariant): a transposed
    # definition fails the off-diagonal finite differences above
    assert np.abs(W - W.T).max() > 1e-3 * np.abs(W).max()


@pytest.mark.parametrize("lmax", [1, 2])
def test_tp_double_backward_is_the_gradient_of_the_vjp(lmax):
    """orc.tp_double_backward (reading A26) pinned through the already pinned first derivative: S(G, V, E, w) = <aV, gV> + <bE, gE> with
    (gV, gE) = orc.tp_backward; central differences of S along random directions of each argument equal <gradient, direction>.
    S is linear in each argument, so the differences are exact up to rounding; a swapped pair of cotangents or a dropped term fails."""
    g = _small_graph("C0")
    rp = g["row_ptr"]
    E, N = g["rvec"].shape[0], rp.shape[0] - 1
    n, dV, dE, P = 3, oracle.dim_v(lmax), oracle.dim_e(lmax), len(oracle.paths(lmax)["l1"])
    rs = np.random.RandomState(5)
    G, V, aV = rs.randn(E, n, dV), rs.randn(E, n, dV), rs.randn(E, n, dV)
    Ee, bE = rs.randn(N, n, dE), rs.randn(N, n, dE)
    w = rs.randn(P)

    def S(G_, V_, E_, w_):
        gV, gE, _ = oracle.tp_backward(lmax, rp, G_, V_, E_, w_, want_gV=True, want_gw=False)
        return float(np.sum(aV * gV) + np.sum(bE * gE))

    dG, dVv, dEe, dw = oracle.tp_double_backward(lmax, rp, G, V, Ee, w, aV, bE)
    h = 1e-3
    scale = abs(S(G, V, Ee, w)) + 1.0
    for name, grad, shape in (("G", dG, G.shape), ("V", dVv, V.shape), ("E", dEe, Ee.shape), ("w", dw, w.shape)):
        d = rs.randn(*shape)
        args_p = dict(G=G, V=V, E=Ee, w=w)
        args_m = dict(args_p)
        args_p[name] = args_p[name] + h * d
        args_m[name] = args_m[name] - h * d
        fd = (S(args_p["G"], args_p["V"], args_p["E"], args_p["w"]) - S(args_m["G"], args_m["V"], args_m["E"], args_m["w"])) / (2 * h)
        assert abs(fd - float(np.sum(grad * d))) <= 1e-9 * scale * 100, (name, fd, float(np.sum(grad * d)))
    # the two cotangents are not interchangeable: zeroing bE leaves dV = 0 and dG = fwd(aV, E)
    dG0, dV0, dE0, _ = oracle.tp_double_backward(lmax, rp, G, V, Ee, w, aV, np.zeros_like(bE))
    assert np.abs(dV0).max() == 0.0
    assert np.allclose(dG0, oracle.tp_forward(lmax, rp, aV, Ee, w), rtol=0, atol=1e-12 * np.abs(dG0).max())


def test_radial_typed_is_radial_per_cutoff_class():
    """oracle.radial_typed (reading A27: a cutoff radius per edge) is the pinned radial() applied per class of edges: with one class it
    is radial() itself, with two classes every edge gets the value radial() gives it at its own cutoff, and the envelope vanishes at
    each edge's own cutoff"""
    g = _small_graph("C0")
    rvec = g["rvec"].astype(np.float64)
    rs = np.random.RandomState(2)
    Wr = rs.randn(5, 8) / np.sqrt(8)
    w0, d0 = oracle.radial(Wr, 4.0, rvec)
    w1, d1 = oracle.radial_typed(Wr, np.full(rvec.shape[0], 4.0), rvec)
    assert np.array_equal(w0, w1) and np.array_equal(d0, d1)
    rce = np.where(np.arange(rvec.shape[0]) % 2 == 0, 4.0, 4.5)
    w2, d2 = oracle.radial_typed(Wr, rce, rvec)
    wa, da = oracle.radial(Wr, 4.0, rvec)
    wb, db = oracle.radial(Wr, 4.5, rvec)
    assert np.array_equal(w2[0::2], wa[0::2]) and np.array_equal(w2[1::2], wb[1::2]) and np.array_equal(d2[1::2], db[1::2])
    edge = np.array([[0.0, 0.0, 4.5 - 1e-9], [0.0, 4.0 - 1e-9, 0.0]])
    wz, _ = oracle.radial_typed(Wr, np.array([4.5, 4.0]), edge)
    assert np.abs(wz).max() < 1e-20

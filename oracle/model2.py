"""Float64 oracle of the two-layer Allegro-style model of BASELINE.json:configs[2] (reading A19, SURVEY 8.c
"Two-layer model for C2"; PAPER.md:85-89 gives only "Allegro layers: 2").

TEST INFRASTRUCTURE, NOT PRODUCT.  Plain PyTorch CPU ops in float64, written in the order of the definition:

    b_e   = [B_b(r_e) u(r_e/r_c)]_{b=1..8}                                 (reading A8)
    x0_e  = W_x0 b_e                                                       (n x 8)
    V0_e[n,(l,(-1)^l),m] = (W_v0 b_e)[n] Y_lm(rhat_e), other-parity slots 0
    for L = 1..n_layers:
        w_e    = W_w[L] x_e                                                (n x n)
        Eenv_i = scale * sum_{e in row i} w_e (x) Y(rhat_e)                (north_star)
        t_p    = C^p (V_e[(l1,p1)], Eenv_c(e)[l2])    per path, channel-wise (north_star)
        V'_e[(l3,p3)] += W_p[L][p] t_p                                     (n x n per path)
        x_e    = u(r_e/r_c) SiLU(A[L] [x_e ; V'_e[:,0e]])   (skipped after the last layer)
    E_tot = sum_e sum_n q[n] V_e[n,0e]                                     (configs[2])

The per-edge gradient g_rvec = dE_tot/dr_e is taken by reverse-mode differentiation of exactly this forward
(torch.autograd, a library primitive), and forces follow from oracle.force_gather.  Pins (tests/test_oracle_model2.py):
central finite differences of E_tot, invariance of E_tot under proper and improper rotations, layer-1 Eenv and
out against the C++ oracle's env_embed / tp_forward (independent loops), sum of forces = 0.
The real CG blocks come from the C++ oracle (oracle.cg_real, Racah + real basis), Y_lm is the Legendre recursion of
SURVEY 8.c step 1 restated with torch ops.
"""
import math

import numpy as np
import torch

import oracle as orc


def sph_harm_torch(lmax, u):
    """real, component-normalised Y_lm at unit vectors u[E,3] -> [E,(lmax+1)^2], index l^2+l+m (reading A1)"""
    x, y, z = u[:, 0], u[:, 1], u[:, 2]
    c = [torch.ones_like(x)]
    s = [torch.zeros_like(x)]
    for m in range(1, lmax + 1):
        c.append(x * c[m - 1] - y * s[m - 1])
        s.append(x * s[m - 1] + y * c[m - 1])
    Q = {}
    for m in range(lmax + 1):
        Q[(m, m)] = torch.full_like(x, float(np.prod(np.arange(2 * m - 1, 0, -2))) if m > 0 else 1.0)
        if m + 1 <= lmax:
            Q[(m + 1, m)] = (2 * m + 1) * z * Q[(m, m)]
        for l in range(m + 2, lmax + 1):
            Q[(l, m)] = ((2 * l - 1) * z * Q[(l - 1, m)] - (l + m - 1) * Q[(l - 2, m)]) / (l - m)
    cols = [None] * (lmax + 1) ** 2
    for l in range(lmax + 1):
        for m in range(0, l + 1):
            K = math.sqrt((2 * l + 1) * math.factorial(l - m) / math.factorial(l + m))
            if m == 0:
                cols[l * l + l] = K * Q[(l, 0)]
            else:
                cols[l * l + l + m] = math.sqrt(2.0) * K * Q[(l, m)] * c[m]
                cols[l * l + l - m] = math.sqrt(2.0) * K * Q[(l, m)] * s[m]
    return torch.stack(cols, dim=1)


def radial_basis_torch(r, rc, nb):
    """[E, nb]: sqrt(2/rc) sin(b pi r/rc)/r * u(r/rc), u(x) = 1 - 28x^6 + 48x^7 - 21x^8; also returns u"""
    x = r / rc
    u = 1.0 - 28.0 * x ** 6 + 48.0 * x ** 7 - 21.0 * x ** 8
    b = torch.arange(1, nb + 1, dtype=r.dtype)
    B = math.sqrt(2.0 / rc) * torch.sin(b[None, :] * math.pi * x[:, None]) / r[:, None]
    return B * u[:, None], u


def feature_offset(l, odd):
    return 2 * l * l + ((2 * l + 1) if odd else 0)


def latent_update(x, s, A, u):
    """scalar latent update between layers (reading A19): z = A [x ; s], x_new = u(r / r_c) SiLU(z); x, s [E, n], A [n, 2n], u [E]"""
    z = torch.cat([x, s], dim=1) @ A.T
    return z, u[:, None] * torch.nn.functional.silu(z)


def forward(params, row_ptr, rvec, taps=None):
    """E_tot (0-d tensor) for rvec [E,3] (float64 tensor, may require grad).  params: lmax, n, nb, n_layers, rc, scale,
    W_x0 [n,nb], W_v0 [n,nb], W_w [L,n,n], W_p [L,P,n,n], A_lat [L-1,n,2n], q [n] (numpy or tensors)."""
    tt = lambda a: torch.as_tensor(np.asarray(a), dtype=torch.float64)
    lmax, n, nb, L = int(params["lmax"]), int(params["n"]), int(params["nb"]), int(params["n_layers"])
    rc, scale = float(params["rc"]), float(params["scale"])
    W_x0, W_v0, W_w, W_p, A_lat, q = (tt(params[k]) for k in ("W_x0", "W_v0", "W_w", "W_p", "A_lat", "q"))
    rp = np.asarray(row_ptr, dtype=np.int64)
    N, E = rp.shape[0] - 1, rvec.shape[0]
    centre = torch.from_numpy(np.repeat(np.arange(N), np.diff(rp)))
    dV, dE = 2 * (lmax + 1) ** 2, (lmax + 1) ** 2
    r = torch.sqrt((rvec * rvec).sum(1))
    Y = sph_harm_torch(lmax, rvec / r[:, None])
    b, u = radial_basis_torch(r, rc, nb)
    x = b @ W_x0.T
    v0 = b @ W_v0.T
    V = torch.zeros((E, n, dV), dtype=torch.float64)
    for l in range(lmax + 1):
        o = feature_offset(l, l % 2 == 1)
        V[:, :, o:o + 2 * l + 1] = v0[:, :, None] * Y[:, None, l * l:l * l + 2 * l + 1]
    paths = orc.paths(lmax)
    P = len(paths["l1"])
    cg = {}
    for layer in range(L):
        w = x @ W_w[layer].T
        Eenv = torch.zeros((N, n, dE), dtype=torch.float64).index_add(0, centre, w[:, :, None] * Y[:, None, :]) * scale
        Ee = Eenv[centre]
        Vn = torch.zeros_like(V)
        for p in range(P):
            l1, l2, l3 = int(paths["l1"][p]), int(paths["l2"][p]), int(paths["l3"][p])
            o1, o2, o3 = int(paths["off1"][p]), int(paths["off2"][p]), int(paths["off3"][p])
            if (l1, l2, l3) not in cg:
                cg[(l1, l2, l3)] = torch.from_numpy(orc.cg_real(l1, l2, l3)[0])
            t = torch.einsum("abm,ena,enb->enm", cg[(l1, l2, l3)], V[:, :, o1:o1 + 2 * l1 + 1], Ee[:, :, o2:o2 + 2 * l2 + 1])
            Vn[:, :, o3:o3 + 2 * l3 + 1] = Vn[:, :, o3:o3 + 2 * l3 + 1] + torch.einsum("on,enm->eom", W_p[layer, p], t)
        if taps is not None:
            taps.append(dict(w=w.detach().numpy(), Eenv=Eenv.detach().numpy(), V_in=V.detach().numpy(), V_out=Vn.detach().numpy(),
                             x_in=x.detach().numpy()))
        if layer < L - 1:
            z, x = latent_update(x, Vn[:, :, 0], A_lat[layer], u)
        V = Vn
    e_edge = (V[:, :, 0] * q[None, :]).sum(1)
    if taps is not None:
        taps.append(dict(e_edge=e_edge.detach().numpy()))
    return e_edge.sum()


def energy_grad(params, row_ptr, rvec, taps=None):
    """-> (E_tot float, g_rvec[E,3] numpy = dE_tot/dr_e)"""
    rv = torch.tensor(np.asarray(rvec, dtype=np.float64), requires_grad=True)
    en = forward(params, row_ptr, rv, taps)
    (g,) = torch.autograd.grad(en, rv)
    return float(en.item()), g.numpy()

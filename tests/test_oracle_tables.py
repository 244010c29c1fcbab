"""Pins for the oracle's tables: complex/real Clebsch-Gordan, path plan, spherical harmonics,
Wigner-D, radial basis.  Everything here compares the oracle with something other than itself:
textbook values (tests/golden), sympy, scipy, closed forms, invariants.  CPU only.
"""
import os

import numpy as np
import pytest
import scipy.special
import sympy
from sympy.physics.quantum.cg import CG

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    for line in open(os.path.join(GOLD, name)):
        line = line.strip()
        if line and not line.startswith("#"):
            yield line.split()


# ------------------------------------------------------------------ complex CG

def test_cg_complex_textbook_values():
    for j1, m1, j2, m2, J, M, sg, num, den in _rows("cg_textbook.txt"):
        exp = (1.0 if sg == "+" else -1.0) * np.sqrt(int(num) / int(den))
        got = oracle.cg_complex(int(j1), int(m1), int(j2), int(m2), int(J), int(M))
        assert abs(got - exp) < 1e-14, (j1, m1, j2, m2, J, M)


@pytest.mark.parametrize("j1,j2", [(0, 0), (1, 0), (1, 1), (2, 1), (1, 2), (2, 2), (3, 1), (3, 2), (2, 3), (3, 3)])
def test_cg_complex_vs_sympy(j1, j2):
    for J in range(abs(j1 - j2), j1 + j2 + 1):
        for m1 in range(-j1, j1 + 1):
            for m2 in range(-j2, j2 + 1):
                M = m1 + m2
                if abs(M) > J:
                    continue
                if (j1 == 3 or j2 == 3) and (m1 + 2 * m2) % 3:      # sample the l=3 blocks
                    continue
                exp = float(CG(j1, m1, j2, m2, J, M).doit())
                assert abs(oracle.cg_complex(j1, m1, j2, m2, J, M) - exp) < 1e-14


def test_cg_complex_unitarity_and_selection():
    for j1 in range(4):
        for j2 in range(4):
            Js = list(range(abs(j1 - j2), j1 + j2 + 1))
            cols = []
            for J in Js:
                for M in range(-J, J + 1):
                    cols.append([oracle.cg_complex(j1, m1, j2, m2, J, M)
                                 for m1 in range(-j1, j1 + 1) for m2 in range(-j2, j2 + 1)])
            A = np.array(cols)
            assert np.allclose(A @ A.T, np.eye(A.shape[0]), atol=1e-14)
    assert oracle.cg_complex(1, 1, 1, 1, 2, 1) == 0.0          # m1+m2 != M
    assert oracle.cg_complex(1, 0, 1, 0, 3, 0) == 0.0          # triangle


# ------------------------------------------------------------------ real CG

def _U(l):
    """complex->real change of basis of reading A1/A2, written from the defining relations
    Y_real(+m) = sqrt2 (-1)^m Re Y_l^m, Y_real(-m) = sqrt2 (-1)^m Im Y_l^m (checked vs scipy below)"""
    U = np.zeros((2 * l + 1, 2 * l + 1), dtype=complex)
    U[l, l] = 1.0
    for m in range(1, l + 1):
        s = (-1.0) ** m
        # Re Y^m = (Y^m + conj Y^m)/2, conj Y^m = (-1)^m Y^{-m}
        U[l + m, l + m] = s / np.sqrt(2)
        U[l + m, l - m] = 1 / np.sqrt(2)
        # Im Y^m = (Y^m - conj Y^m)/(2i)
        U[l - m, l + m] = s / (1j * np.sqrt(2))
        U[l - m, l - m] = -1 / (1j * np.sqrt(2))
    return U


def _Y_scipy_real(l, rhat):
    x, y, z = rhat
    theta, phi = np.arccos(z), np.arctan2(y, x)
    Yc = np.array([scipy.special.sph_harm_y(l, m, theta, phi) for m in range(-l, l + 1)])
    Yr = _U(l) @ Yc * np.sqrt(4 * np.pi)
    assert np.abs(Yr.imag).max() < 1e-13
    return Yr.real


def test_real_cg_from_sympy_and_scipy_checked_basis():
    """C = Re T + Im T with T built here from sympy's complex CG and the basis change U that the
    scipy check above validates.  Covers every triangle up to l = 2 and the mixed l = 3 ones."""
    tris = [(a, b, c) for a in range(3) for b in range(3) for c in range(abs(a - b), min(a + b, 3) + 1)]
    tris += [(3, 1, 2), (1, 3, 3), (3, 3, 0), (3, 2, 1), (3, 3, 1)]
    for l1, l2, l3 in tris:
        U1, U2, U3 = _U(l1), _U(l2), _U(l3)
        cg = np.zeros((2 * l1 + 1, 2 * l2 + 1, 2 * l3 + 1))
        for a in range(-l1, l1 + 1):
            for b in range(-l2, l2 + 1):
                if abs(a + b) <= l3:
                    cg[a + l1, b + l2, a + b + l3] = float(CG(l1, a, l2, b, l3, a + b).doit())
        T = np.einsum("ax,by,cz,xyz->abc", U1.conj(), U2.conj(), U3, cg)
        C, mre, mim = oracle.cg_real(l1, l2, l3)
        if (l1 + l2 + l3) % 2 == 0:
            assert np.abs(T.imag).max() < 1e-14 and mim < 1e-14
        else:
            assert np.abs(T.real).max() < 1e-14 and mre < 1e-14
        assert np.allclose(C, T.real + T.imag, atol=1e-14), (l1, l2, l3)


def test_real_cg_orthonormal_all_triangles():
    for l1 in range(4):
        for l2 in range(4):
            for l3 in range(abs(l1 - l2), min(l1 + l2, 3) + 1):
                C, _, _ = oracle.cg_real(l1, l2, l3)
                G = np.einsum("abM,abN->MN", C, C)
                assert np.allclose(G, np.eye(2 * l3 + 1), atol=1e-14)
                assert abs((C ** 2).sum() - (2 * l3 + 1)) < 1e-13


def test_real_cg_special_values():
    C110, _, _ = oracle.cg_real(1, 1, 0)
    assert np.allclose(C110[:, :, 0], -np.eye(3) / np.sqrt(3), atol=1e-15)
    C111, _, _ = oracle.cg_real(1, 1, 1)
    rs = np.random.RandomState(0)
    yzx = lambda v: np.array([v[1], v[2], v[0]])
    for _ in range(5):
        a, b = rs.randn(3), rs.randn(3)
        got = np.einsum("abc,a,b->c", C111, yzx(a), yzx(b))
        assert np.allclose(got, yzx(np.cross(a, b)) / np.sqrt(2), atol=1e-14)
    C000, _, _ = oracle.cg_real(0, 0, 0)
    assert abs(C000[0, 0, 0] - 1.0) < 1e-15
    for l in range(1, 4):    # coupling with a scalar is the identity
        C, _, _ = oracle.cg_real(l, 0, l)
        assert np.allclose(C[:, 0, :], np.eye(2 * l + 1), atol=1e-15)
        C, _, _ = oracle.cg_real(0, l, l)
        assert np.allclose(C[0, :, :], np.eye(2 * l + 1), atol=1e-15)


def test_gaunt_relation():
    """C^{l1 l2 l3} (Y_l1 (x) Y_l2) = kappa Y_l3 on the same unit vector; zero for odd l1+l2+l3."""
    rs = np.random.RandomState(1)
    kap = {(int(a), int(b), int(c)): float(k) for a, b, c, k in _rows("gaunt_kappa.txt")}
    for l1 in range(4):
        for l2 in range(4):
            for l3 in range(abs(l1 - l2), min(l1 + l2, 3) + 1):
                C, _, _ = oracle.cg_real(l1, l2, l3)
                for _ in range(3):
                    r = rs.randn(3)
                    Y, _ = oracle.sph_harm(3, r)
                    y = lambda l: Y[l * l:(l + 1) ** 2]
                    lhs = np.einsum("abc,a,b->c", C, y(l1), y(l2))
                    if (l1 + l2 + l3) % 2:
                        assert np.abs(lhs).max() < 1e-13
                    else:
                        k = np.sqrt((2 * l1 + 1) * (2 * l2 + 1) / (2 * l3 + 1)) * float(CG(l1, 0, l2, 0, l3, 0).doit())
                        if (l1, l2, l3) in kap:
                            assert abs(k - kap[(l1, l2, l3)]) < 1e-14
                        assert np.allclose(lhs, k * y(l3), atol=1e-13), (l1, l2, l3)


# ------------------------------------------------------------------ path plan

def test_path_plan_counts_and_order():
    for lmax, P, nnz, half in [(1, 10, 32, 16), (2, 30, 274, 137), (3, 68, 1222, 611)]:
        p = oracle.paths(lmax)
        assert len(p["l1"]) == P
        L = oracle.cg_list(lmax)
        assert len(L["coef"]) == nnz
        assert int((p["p1"][L["path"]] == 0).sum()) == half           # per parity half
        keys = list(zip(p["l1"], p["p1"], p["l2"], p["l3"]))
        assert keys == sorted(keys) and len(set(keys)) == P
        for t in range(P):
            l1, p1, l2, l3, p3 = (int(p[k][t]) for k in ("l1", "p1", "l2", "l3", "p3"))
            assert abs(l1 - l2) <= l3 <= min(l1 + l2, lmax)
            assert p3 == (p1 + l2) % 2                                # p3 = p1 (-1)^l2
            assert p["off1"][t] == 2 * l1 * l1 + (2 * l1 + 1 if p1 else 0)
            assert p["off2"][t] == l2 * l2
            assert p["off3"][t] == 2 * l3 * l3 + (2 * l3 + 1 if p3 else 0)
        # sorted (path, i, j, k), entries inside their blocks, values equal the dense blocks
        q = list(zip(L["path"], L["i"], L["j"], L["k"]))
        assert q == sorted(q) and len(set(q)) == nnz
        for t in range(0, nnz, 7):
            pa = int(L["path"][t])
            C, _, _ = oracle.cg_real(int(p["l1"][pa]), int(p["l2"][pa]), int(p["l3"][pa]))
            assert C[L["i"][t] - p["off1"][pa], L["j"][t] - p["off2"][pa], L["k"][t] - p["off3"][pa]] == L["coef"][t]
        # every path is represented; every (V comp, Eenv comp) pair couples to something
        assert set(L["path"]) == set(range(P))
        assert len(set(zip(L["i"], L["j"]))) == oracle.dim_v(lmax) * oracle.dim_e(lmax)
    assert oracle.dim_v(2) == 18 and oracle.dim_e(2) == 9 and oracle.dim_v(3) == 32


# ------------------------------------------------------------------ spherical harmonics

def _closed_forms(r):
    x, y, z = r / np.linalg.norm(r)
    s3, s5, s7, s15 = np.sqrt(3), np.sqrt(5), np.sqrt(7), np.sqrt(15)
    return np.array([
        1.0,
        s3 * y, s3 * z, s3 * x,
        s15 * x * y, s15 * y * z, s5 / 2 * (3 * z * z - 1), s15 * x * z, s15 / 2 * (x * x - y * y),
        np.sqrt(35 / 8) * y * (3 * x * x - y * y), np.sqrt(105) * x * y * z, np.sqrt(21 / 8) * y * (5 * z * z - 1),
        s7 / 2 * z * (5 * z * z - 3), np.sqrt(21 / 8) * x * (5 * z * z - 1), np.sqrt(105) / 2 * z * (x * x - y * y),
        np.sqrt(35 / 8) * x * (x * x - 3 * y * y)])


def test_sph_harm_closed_forms_and_scipy():
    rs = np.random.RandomState(2)
    pts = [rs.randn(3) * rs.uniform(0.5, 6) for _ in range(20)] + [np.array([0, 0, 2.0]), np.array([1.0, 0, 0]),
                                                                     np.array([0, -3.0, 0]), np.array([0, 0, -1.0])]
    for r in pts:
        Y, _ = oracle.sph_harm(3, r)
        assert np.allclose(Y, _closed_forms(r), atol=1e-14)
        for l in range(4):
            assert abs((Y[l * l:(l + 1) ** 2] ** 2).sum() - (2 * l + 1)) < 1e-13
        rh = r / np.linalg.norm(r)
        if abs(rh[2]) < 1 - 1e-9:
            for l in range(4):
                assert np.allclose(Y[l * l:(l + 1) ** 2], _Y_scipy_real(l, rh), atol=1e-13)
        # lower lmax is a prefix
        Y2, _ = oracle.sph_harm(2, r)
        assert np.array_equal(Y2, Y[:9])


def test_sph_harm_addition_theorem():
    rs = np.random.RandomState(3)
    for _ in range(10):
        a, b = rs.randn(3), rs.randn(3)
        Ya, _ = oracle.sph_harm(3, a)
        Yb, _ = oracle.sph_harm(3, b)
        c = a @ b / np.linalg.norm(a) / np.linalg.norm(b)
        for l in range(4):
            Pl = scipy.special.eval_legendre(l, c)
            assert abs(Ya[l * l:(l + 1) ** 2] @ Yb[l * l:(l + 1) ** 2] - (2 * l + 1) * Pl) < 1e-13


def test_sph_harm_derivative():
    rs = np.random.RandomState(4)
    for _ in range(10):
        r = rs.randn(3) * rs.uniform(0.9, 6)
        _, dY = oracle.sph_harm(3, r)
        assert np.abs(dY @ r).max() < 1e-13                      # Euler: degree-0 homogeneous
        h = 1e-6 * np.linalg.norm(r)
        for a in range(3):
            e = np.zeros(3)
            e[a] = h
            fd = (oracle.sph_harm(3, r + e)[0] - oracle.sph_harm(3, r - e)[0]) / (2 * h)
            assert np.allclose(dY[:, a], fd, atol=2e-9)


# ------------------------------------------------------------------ Wigner D

def test_wigner_D_matches_least_squares_fit_and_group_law():
    rs = np.random.RandomState(5)
    for _ in range(4):
        a, b, g = rs.uniform(0, 2 * np.pi), rs.uniform(0, np.pi), rs.uniform(0, 2 * np.pi)
        R = oracle.rotation_matrix(a, b, g)
        assert np.allclose(R @ R.T, np.eye(3), atol=1e-15) and abs(np.linalg.det(R) - 1) < 1e-14
        pts = rs.randn(60, 3)
        Y0 = np.array([oracle.sph_harm(3, p)[0] for p in pts])
        Y1 = np.array([oracle.sph_harm(3, R @ p)[0] for p in pts])
        for l in range(4):
            sl = slice(l * l, (l + 1) ** 2)
            fit = np.linalg.lstsq(Y0[:, sl], Y1[:, sl], rcond=None)[0].T      # Y1 = D Y0
            D = oracle.wigner_D_real(l, a, b, g)
            assert np.allclose(D, fit, atol=1e-12), l
            assert np.allclose(D @ D.T, np.eye(2 * l + 1), atol=1e-13)
    # homomorphism: D(Rz(a1)) D(Rz(a2)) = D(Rz(a1+a2)), and a general product through the fit
    for l in range(1, 4):
        assert np.allclose(oracle.wigner_D_real(l, 0.3, 0, 0) @ oracle.wigner_D_real(l, 0.5, 0, 0),
                           oracle.wigner_D_real(l, 0.8, 0, 0), atol=1e-14)
        assert np.allclose(oracle.wigner_D_real(l, 0, 0.4, 0) @ oracle.wigner_D_real(l, 0, 0.7, 0),
                           oracle.wigner_D_real(l, 0, 1.1, 0), atol=1e-14)
        assert np.allclose(oracle.wigner_D_real(l, 0.2, 0.4, 0.9),
                           oracle.wigner_D_real(l, 0.2, 0, 0) @ oracle.wigner_D_real(l, 0, 0.4, 0)
                           @ oracle.wigner_D_real(l, 0, 0, 0.9), atol=1e-14)


def test_wigner_small_d_vs_sympy():
    from sympy.physics.quantum.spin import Rotation
    beta = 0.7
    for l in (1, 2):
        # real-basis D for a pure y-rotation, rebuilt from sympy's small d and the checked U
        d = np.array([[complex(sympy.N(Rotation.d(l, mp, m, beta).doit())).real for m in range(-l, l + 1)]
                      for mp in range(-l, l + 1)])
        U = _U(l)
        D = (U @ d.conj() @ U.conj().T).real
        assert np.allclose(D, oracle.wigner_D_real(l, 0.0, beta, 0.0), atol=1e-13)


# ------------------------------------------------------------------ radial

def _u_general(x, p=6):
    return 1 - (p + 1) * (p + 2) / 2 * x ** p + p * (p + 2) * x ** (p + 1) - p * (p + 1) / 2 * x ** (p + 2)


def test_radial_basis_and_cutoff():
    rc = 6.0
    Wr = np.eye(8)
    r = np.linspace(1e-4, rc * (1 - 1e-9), 200001)
    rvec = np.zeros((r.size, 3))
    rvec[:, 2] = r
    w, dw = oracle.radial(Wr, rc, rvec)
    x = r / rc
    u = _u_general(x)
    # functional form of B_b: ratios of basis functions
    assert np.allclose(w[:, 2] * np.sin(np.pi * x), w[:, 0] * np.sin(3 * np.pi * x), atol=1e-12)
    # cutoff envelope: w_1 r / (sqrt(2/rc) sin(pi x)) = u(x)
    mid = slice(1000, -1000)
    env = w[mid, 0] * r[mid] / (np.sqrt(2 / rc) * np.sin(np.pi * x[mid]))
    assert np.allclose(env, u[mid], atol=1e-12)
    assert abs(_u_general(0.0) - 1) < 1e-15 and abs(_u_general(1.0)) < 1e-12
    h = 1e-3
    assert abs(_u_general(1 - h) / h ** 3 - 56.0) < 0.5          # u = u' = u'' = 0 at x = 1, u''' = -336
    # orthonormality of the bare Bessel functions: int_0^rc B_a B_b r^2 dr = delta_ab
    B = w[mid] / u[mid, None]
    rr = r[mid]
    gram = np.trapezoid(B[:, :, None] * B[:, None, :] * (rr ** 2)[:, None, None], rr, axis=0)
    assert np.allclose(gram, np.eye(8), atol=2e-3)
    # derivative
    k = np.arange(5000, r.size - 5000, 9973)
    hh = 1e-6
    rp = rvec[k].copy()
    rm = rvec[k].copy()
    rp[:, 2] += hh
    rm[:, 2] -= hh
    fd = (oracle.radial(Wr, rc, rp)[0] - oracle.radial(Wr, rc, rm)[0]) / (2 * hh)
    assert np.allclose(dw[k], fd, atol=1e-8)
    # general linear map and direction independence
    rs = np.random.RandomState(6)
    W = rs.randn(5, 8)
    v = rs.randn(50, 3)
    v *= (rs.uniform(0.9, 5.9, 50) / np.linalg.norm(v, axis=1))[:, None]
    w2, _ = oracle.radial(W, rc, v)
    vz = np.zeros_like(v)
    vz[:, 2] = np.linalg.norm(v, axis=1)
    w3, _ = oracle.radial(np.eye(8), rc, vz)
    assert np.allclose(w2, w3 @ W.T, atol=1e-13)

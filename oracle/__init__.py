"""ctypes loader for the float64 CPU oracle (oracle/allegro_oracle.cpp).

TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
CPU-baseline legs (cpu_baseline, --impl reference) may import this package.  The product
package paper_2504_16068_b200 never imports it and shares no code with it.

Thin numpy marshalling only; all arithmetic is in the C++ file, each function of which cites
the passage (PAPER.md line / DESIGN.md reading) it follows.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRCS = ["allegro_oracle.cpp"]
_LIB = os.path.join(_HERE, "liballegro_oracle.so")
_lib = None


def build(force=False):
    """g++ -O2, no intrinsics, no OpenMP."""
    srcs = [os.path.join(_HERE, s) for s in _SRCS if os.path.exists(os.path.join(_HERE, s))]
    deps = srcs + [os.path.join(_HERE, "allegro_oracle.h")]
    if not force and os.path.exists(_LIB) and all(os.path.getmtime(_LIB) >= os.path.getmtime(d) for d in deps):
        return _LIB
    tmp = _LIB + ".tmp.%d" % os.getpid()
    cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-o", tmp] + srcs
    subprocess.check_call(cmd)
    os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _declare(_lib)
    return _lib


_i32p = C.POINTER(C.c_int32)
_f64p = C.POINTER(C.c_double)


def _declare(L):
    L.orc_cg_complex.restype = C.c_double
    L.orc_cg_complex.argtypes = [C.c_int] * 6
    L.orc_nnz.restype = C.c_int64
    L.orc_segments.restype = C.c_int64


def _d(a):
    return None if a is None else a.ctypes.data_as(_f64p)


def _i(a):
    return None if a is None else a.ctypes.data_as(_i32p)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def dim_v(lmax):
    return lib().orc_dim_v(C.c_int(lmax))


def dim_e(lmax):
    return lib().orc_dim_e(C.c_int(lmax))


def cg_complex(j1, m1, j2, m2, j3, m3):
    return lib().orc_cg_complex(j1, m1, j2, m2, j3, m3)


def cg_real(l1, l2, l3):
    """-> (C[2l1+1, 2l2+1, 2l3+1], max|Re T|, max|Im T|)"""
    out = np.zeros((2 * l1 + 1, 2 * l2 + 1, 2 * l3 + 1))
    re, im = C.c_double(), C.c_double()
    lib().orc_cg_real(l1, l2, l3, _d(out), C.byref(re), C.byref(im))
    return out, re.value, im.value


def paths(lmax):
    P = lib().orc_num_paths(lmax)
    names = ["l1", "p1", "l2", "l3", "p3", "off1", "off2", "off3"]
    arrs = [np.zeros(P, dtype=np.int32) for _ in names]
    lib().orc_paths(lmax, *[_i(a) for a in arrs])
    return dict(zip(names, arrs))


def cg_list(lmax):
    nnz = lib().orc_nnz(lmax)
    path, i, j, k = [np.zeros(nnz, dtype=np.int32) for _ in range(4)]
    coef = np.zeros(nnz)
    lib().orc_cg_list(lmax, _i(path), _i(i), _i(j), _i(k), _d(coef))
    return dict(path=path, i=i, j=j, k=k, coef=coef)


def sph_harm(lmax, r):
    """-> (Y[dE], dYdr[dE,3])"""
    r = _f64(r)
    dE = (lmax + 1) ** 2
    Y = np.zeros(dE)
    dY = np.zeros((dE, 3))
    lib().orc_sph_harm(lmax, _d(r), _d(Y), _d(dY))
    return Y, dY


def rotation_matrix(alpha, beta, gamma):
    R = np.zeros((3, 3))
    lib().orc_rotation_matrix(C.c_double(alpha), C.c_double(beta), C.c_double(gamma), _d(R))
    return R


def wigner_D_real(l, alpha, beta, gamma):
    D = np.zeros((2 * l + 1, 2 * l + 1))
    lib().orc_wigner_D_real(l, C.c_double(alpha), C.c_double(beta), C.c_double(gamma), _d(D))
    return D


def radial(Wr, rc, rvec):
    """-> (w[E,n], dwdr[E,n])"""
    Wr = _f64(Wr)
    rvec = _f64(rvec)
    n, nb = Wr.shape
    E = rvec.shape[0]
    w = np.zeros((E, n))
    dw = np.zeros((E, n))
    lib().orc_radial(n, nb, C.c_double(rc), _d(Wr), C.c_int64(E), _d(rvec), _d(w), _d(dw))
    return w, dw


def radial_typed(Wr, rc_edge, rvec):
    """radial() with a cutoff radius per edge (per-edge-type cutoffs, reading A27): the pinned orc_radial evaluated on the edges of
    every distinct cutoff value in turn -> (w [E,n], dwdr [E,n])"""
    rc_edge = np.asarray(rc_edge, dtype=np.float64)
    rvec = _f64(rvec)
    w = np.zeros((rvec.shape[0], np.asarray(Wr).shape[0]))
    dw = np.zeros_like(w)
    for rc in np.unique(rc_edge):
        m = rc_edge == rc
        w[m], dw[m] = radial(Wr, float(rc), rvec[m])
    return w, dw


def radial_backward(rvec, g_w, dwdr, g_rvec):
    """g_rvec += (sum_n g_w dwdr) rhat, in place; returns g_rvec"""
    rvec, g_w, dwdr = _f64(rvec), _f64(g_w), _f64(dwdr)
    assert g_rvec.dtype == np.float64 and g_rvec.flags.c_contiguous
    E, n = g_w.shape
    lib().orc_radial_backward(n, C.c_int64(E), _d(rvec), _d(g_w), _d(dwdr), _d(g_rvec))
    return g_rvec


def segments(row_ptr, T):
    row_ptr = _i32(row_ptr)
    N = row_ptr.shape[0] - 1
    cnt = lib().orc_segments(_i(row_ptr), N, T, None, C.c_int64(0))
    items = np.zeros((cnt, 3), dtype=np.int32)
    lib().orc_segments(_i(row_ptr), N, T, _i(items), C.c_int64(cnt))
    return items


def env_embed(lmax, row_ptr, rvec, w, scale=1.0):
    row_ptr, rvec, w = _i32(row_ptr), _f64(rvec), _f64(w)
    N = row_ptr.shape[0] - 1
    n = w.shape[1]
    Eenv = np.zeros((N, n, dim_e(lmax)))
    lib().orc_env_embed(lmax, n, N, _i(row_ptr), _d(rvec), _d(w), C.c_double(scale), _d(Eenv))
    return Eenv


def _crange(row_ptr, centres):
    N = row_ptr.shape[0] - 1
    return (0, N) if centres is None else (int(centres[0]), int(centres[1]))


def tp_forward(lmax, row_ptr, V, Eenv, path_w, variant="sparse", centres=None, out=None):
    """wmode is inferred from path_w.ndim (1: scalar per path, 3: dense [P,n,n])."""
    row_ptr, V, Eenv, path_w = _i32(row_ptr), _f64(V), _f64(Eenv), _f64(path_w)
    N = row_ptr.shape[0] - 1
    n = V.shape[1]
    wmode = 0 if path_w.ndim == 1 else 1
    if out is None:
        out = np.zeros_like(V)
    c_lo, c_hi = _crange(row_ptr, centres)
    fn = lib().orc_tp_forward_sparse if variant == "sparse" else lib().orc_tp_forward_dense
    fn(lmax, n, wmode, N, _i(row_ptr), c_lo, c_hi, _d(V), _d(Eenv), _d(path_w), _d(out))
    return out


def tp_backward(lmax, row_ptr, G, V, Eenv, path_w, want_gV=True, want_gw=True, centres=None):
    """-> (gV or None, gEenv, g_path_w or None)"""
    row_ptr, G, V, Eenv, path_w = _i32(row_ptr), _f64(G), _f64(V), _f64(Eenv), _f64(path_w)
    N = row_ptr.shape[0] - 1
    n = V.shape[1]
    wmode = 0 if path_w.ndim == 1 else 1
    gV = np.zeros_like(V) if want_gV else None
    gE = np.zeros_like(Eenv)
    gw = np.zeros_like(path_w) if want_gw else None
    c_lo, c_hi = _crange(row_ptr, centres)
    lib().orc_tp_backward(lmax, n, wmode, N, _i(row_ptr), c_lo, c_hi, _d(G), _d(V), _d(Eenv), _d(path_w),
                          _d(gV), _d(gE), _d(gw))
    return gV, gE, gw


def env_embed_backward(lmax, row_ptr, gEenv, rvec, w, scale=1.0, centres=None):
    """-> (g_rvec[E,3], g_w[E,n])"""
    row_ptr, gEenv, rvec, w = _i32(row_ptr), _f64(gEenv), _f64(rvec), _f64(w)
    N = row_ptr.shape[0] - 1
    n = w.shape[1]
    g_r = np.zeros_like(rvec)
    g_w = np.zeros_like(w)
    c_lo, c_hi = _crange(row_ptr, centres)
    lib().orc_env_embed_backward(lmax, n, N, _i(row_ptr), c_lo, c_hi, _d(gEenv), _d(rvec), _d(w),
                                 C.c_double(scale), _d(g_r), _d(g_w))
    return g_r, g_w


def force_gather(row_ptr, rev, g_rvec):
    row_ptr, rev, g_rvec = _i32(row_ptr), _i32(rev), _f64(g_rvec)
    N = row_ptr.shape[0] - 1
    F = np.zeros((N, 3))
    lib().orc_force_gather(N, _i(row_ptr), _i(rev), _d(g_rvec), _d(F))
    return F


def tp_double_backward(lmax, row_ptr, G, V, Eenv, path_w, aV, bE):
    """gradients of S = <aV, gV> + <bE, gEenv> (outputs of tp_backward, scalar weights) -> (dG, dV, dEenv, dw)  (reading A26)"""
    row_ptr, G, V, Eenv, path_w, aV, bE = _i32(row_ptr), _f64(G), _f64(V), _f64(Eenv), _f64(path_w), _f64(aV), _f64(bE)
    assert path_w.ndim == 1
    N, n = row_ptr.shape[0] - 1, V.shape[1]
    dG, dV, dE, dw = np.zeros_like(V), np.zeros_like(V), np.zeros_like(Eenv), np.zeros_like(path_w)
    lib().orc_tp_double_backward(lmax, n, N, _i(row_ptr), _d(G), _d(V), _d(Eenv), _d(path_w), _d(aV), _d(bE), _d(dG), _d(dV), _d(dE), _d(dw))
    return dG, dV, dE, dw


def virial(rvec, g_rvec):
    """W[a][b] = sum_e g_rvec[e][a] rvec[e][b] (reading A25) -> [3,3]"""
    rvec, g_rvec = _f64(rvec), _f64(g_rvec)
    W = np.zeros((3, 3))
    lib().orc_virial(C.c_int64(rvec.shape[0]), _d(rvec), _d(g_rvec), _d(W))
    return W


def edge_energy(lmax, out, q, kappa, want_G=True):
    """-> (e_edge[E], G or None)"""
    out, q = _f64(out), _f64(q)
    E, n, _ = out.shape
    e_edge = np.zeros(E)
    G = np.zeros_like(out) if want_G else None
    lib().orc_edge_energy(lmax, n, C.c_int64(E), _d(out), _d(q), C.c_double(kappa), _d(e_edge), _d(G))
    return e_edge, G


def segment_sum(ptr, vals):
    ptr, vals = _i32(ptr), _f64(vals)
    nseg = ptr.shape[0] - 1
    out = np.zeros(nseg)
    lib().orc_segment_sum(_i(ptr), nseg, _d(vals), _d(out))
    return out

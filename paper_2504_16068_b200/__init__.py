"""paper_2504_16068_b200 -- Python binding of liballegro_b200.so (include/allegro_b200.h).

Argument marshalling only: every step of the hot path runs in the library's CUDA kernels (sm_100a).
torch is used for device memory and streams.  There is no CPU fallback and nothing here imports the
oracle: if the shared library is missing the import of any entry point raises.

Names mirror the C ABI without the `allegro_` prefix:
    Plan(l_max, n, dtype, wmode)            allegro_plan_create / _destroy / _paths / _cg
    segments_build, env_embed, tp_forward, tp_forward_energy, tp_backward, env_embed_backward, force_gather,
    radial_forward, radial_backward, edge_energy, segment_sum, launch_count
"""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liballegro_b200.so")
_lib = None

F32, F64 = 0, 1
W_SCALAR, W_DENSE = 0, 1
_STATUS = {0: "ALLEGRO_OK", 1: "ALLEGRO_EINVAL", 2: "ALLEGRO_EUNSUPPORTED", 3: "ALLEGRO_ECUDA", 4: "ALLEGRO_ENOMEM"}

_vp, _i32p, _f64p = C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_double)

# name -> (restype, argtypes); one row per symbol declared in include/allegro_b200.h
SIGNATURES = {
    "allegro_plan_create": (C.c_int, [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(_vp)]),
    "allegro_plan_destroy": (None, [_vp]),
    "allegro_plan_bind_weights": (C.c_int, [_vp, _vp, _vp]),
    "allegro_plan_set_out_blocks": (C.c_int, [_vp, C.c_uint]),
    "allegro_plan_set_in_blocks": (C.c_int, [_vp, C.c_uint]),
    "allegro_plan_num_paths": (C.c_int, [_vp]),
    "allegro_plan_dim_v": (C.c_int, [_vp]),
    "allegro_plan_dim_e": (C.c_int, [_vp]),
    "allegro_plan_nnz": (C.c_long, [_vp]),
    "allegro_plan_paths": (C.c_int, [_vp] + [_i32p] * 8),
    "allegro_plan_cg": (C.c_int, [_vp] + [_i32p] * 4 + [_f64p]),
    "allegro_cg_real_block": (C.c_int, [C.c_int, C.c_int, C.c_int, _f64p]),
    "allegro_segments_build": (C.c_int, [_i32p, C.c_int, C.c_int, _i32p, C.c_long, C.POINTER(C.c_long)]),
    "allegro_env_embed": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, C.c_long, _vp, _vp, C.c_double, _vp, _vp, C.c_size_t, _vp]),
    "allegro_tp_forward": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, C.c_long, _vp, _vp, _vp, _vp, _vp]),
    "allegro_tp_forward_aux": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, C.c_long, _vp, _vp, _vp, _vp, _vp, _vp]),
    "allegro_tp_backward_aux": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, C.c_long, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, C.c_size_t, _vp]),
    "allegro_tp_forward_outer": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, C.c_long, _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "allegro_tp_backward_outer": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, C.c_long, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, C.c_size_t,
                                            _vp]),
    "allegro_edge_embed_factors": (C.c_int, [_vp, C.c_long, _vp, _vp, _vp, C.c_int, C.c_double, _vp, _vp, _vp]),
    "allegro_edge_embed_factors_backward": (C.c_int, [_vp, C.c_long, _vp, _vp, _vp, C.c_int, C.c_double, _vp, _vp, _vp, _vp, _vp]),
    "allegro_tp_forward_energy": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, C.c_long, _vp, _vp, _vp, _vp, C.c_double, _vp, _vp, _vp, _vp]),
    "allegro_tp_backward": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, C.c_long, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, C.c_size_t, _vp]),
    "allegro_tp_backward_energy": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, C.c_long, _vp, _vp, _vp, _vp, _vp, C.c_double, _vp, _vp, _vp, _vp,
                                             C.c_size_t, _vp]),
    "allegro_tp_fused_energy": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, C.c_long, _vp, _vp, _vp, _vp, C.c_double, _vp, _vp, _vp, _vp, _vp,
                                          C.c_size_t, _vp]),
    "allegro_tp_double_backward_workspace": (C.c_size_t, [_vp, C.c_int, C.c_long]),
    "allegro_tp_double_backward": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, C.c_size_t, _vp]),
    "allegro_tp_backward_workspace": (C.c_size_t, [_vp, C.c_int, C.c_long, C.c_long, C.c_int]),
    "allegro_tp_backward_static_capacity": (C.c_size_t, []),
    "allegro_tp_backward_static": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, C.c_long, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "allegro_env_workspace": (C.c_size_t, [_vp, C.c_int, C.c_long]),
    "allegro_env_embed_backward": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, _vp, _vp, C.c_double, _vp, _vp, _vp]),
    "allegro_force_gather": (C.c_int, [C.c_int, C.c_long, _vp, _vp, _vp, C.c_int, _vp, _vp]),
    "allegro_radial_forward": (C.c_int, [C.c_int, C.c_int, C.c_double, C.c_int, C.c_long, _vp, _vp, _vp, _vp]),
    "allegro_radial_backward": (C.c_int, [C.c_int, C.c_int, C.c_double, C.c_int, C.c_long, _vp, _vp, _vp, _vp, _vp]),
    "allegro_env_radial_forward": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, C.c_long, _vp, _vp, C.c_int, C.c_double, C.c_double, _vp, _vp, _vp,
                                             C.c_size_t, _vp]),
    "allegro_env_radial_backward": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, _vp, _vp, C.c_int, C.c_double, C.c_double, _vp, _vp, _vp]),
    "allegro_edge_energy": (C.c_int, [_vp, C.c_long, _vp, _vp, C.c_double, _vp, _vp, _vp]),
    "allegro_segment_sum": (C.c_int, [_vp, C.c_int, _vp, C.c_int, _vp, _vp]),
    "allegro_virial": (C.c_int, [C.c_long, _vp, _vp, C.c_int, _vp, _vp]),
    "allegro_check_graph": (C.c_int, [C.c_int, C.c_long, _vp, _vp, C.c_long, _vp, _vp, _vp, C.c_int, C.POINTER(C.c_long), _vp]),
    "allegro_layer_step_host_workspace": (C.c_size_t, [_vp, C.c_int, C.c_long, C.c_int, C.c_int]),
    "allegro_layer_step_host": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, _vp, _vp, _vp, C.c_int, C.c_double, _vp, _vp, C.c_double, C.c_double,
                                          C.c_int, _vp, _vp, _vp, C.c_size_t, _vp]),
    "allegro_layer_step_workspace": (C.c_size_t, [_vp, C.c_int, C.c_long, C.c_int]),
    "allegro_layer_step_create": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, _vp, _vp, _vp, C.c_int, C.c_double, _vp, C.c_double, C.c_double, C.c_int,
                                            _vp, _vp, _vp, C.c_size_t, C.POINTER(_vp)]),
    "allegro_layer_step_launch": (C.c_int, [_vp, _vp]),
    "allegro_layer_step_buffer": (_vp, [_vp, C.c_char_p]),
    "allegro_layer_step_num_kernels": (C.c_int, [_vp]),
    "allegro_layer_step_destroy": (None, [_vp]),
    "allegro_edge_embed": (C.c_int, [_vp, C.c_long, _vp, _vp, _vp, C.c_int, C.c_double, _vp, _vp, _vp]),
    "allegro_edge_embed_backward": (C.c_int, [_vp, C.c_long, _vp, _vp, _vp, C.c_int, C.c_double, _vp, _vp, _vp, _vp]),
    "allegro_linear": (C.c_int, [C.c_long, C.c_int, C.c_int, C.c_int, _vp, _vp, C.c_int, C.c_int, _vp, _vp]),
    "allegro_latent_forward": (C.c_int, [C.c_long, C.c_int, C.c_int, C.c_double, C.c_int, _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "allegro_latent_backward": (C.c_int, [C.c_long, C.c_int, C.c_int, C.c_double, C.c_int, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "allegro_add_inplace": (C.c_int, [C.c_long, C.c_int, _vp, _vp, _vp]),
    "allegro_neighbour_workspace": (C.c_size_t, [C.c_int]),
    "allegro_neighbour_count": (C.c_int, [C.c_int, _vp, C.c_double, _f64p, _f64p, C.c_double, _vp, _vp, C.c_int, _vp, _vp, _vp, C.c_size_t, _vp,
                                          C.POINTER(C.c_long)]),
    "allegro_neighbour_fill": (C.c_int, [C.c_int, _vp, C.c_double, _f64p, _f64p, C.c_double, _vp, _vp, C.c_int, _vp, _vp, C.c_long, _vp, _vp, _vp, _vp,
                                         C.c_int, _vp, C.c_size_t, _vp]),
    "allegro_env_linear_forward": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, _vp, _vp, C.c_int, C.c_double, _vp, _vp]),
    "allegro_env_linear_backward": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, _vp, _vp, _vp, C.c_int, C.c_double, _vp, C.c_int, _vp, C.c_int, _vp]),
    "allegro_env_radial_forward_typed": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, C.c_long, _vp, _vp, C.c_int, _vp, C.c_double, _vp, _vp, _vp,
                                                   C.c_size_t, _vp]),
    "allegro_env_radial_backward_typed": (C.c_int, [_vp, C.c_int, C.c_long, _vp, _vp, _vp, _vp, C.c_int, _vp, C.c_double, _vp, _vp, _vp]),
    "allegro_measure_fp32_fma_peak": (C.c_int, [_vp, C.POINTER(C.c_double)]),
    "allegro_measure_tf32_mma_peak": (C.c_int, [_vp, C.POINTER(C.c_double)]),
    "allegro_measure_tf32_mma_rate": (C.c_int, [C.c_int, _vp, C.POINTER(C.c_double)]),
    "allegro_status_str": (C.c_char_p, [C.c_int]),
    "allegro_last_error": (C.c_char_p, []),
    "allegro_launch_count": (C.c_long, []),
}


class AllegroError(RuntimeError):
    def __init__(self, status, detail):
        super().__init__("%s: %s" % (_STATUS.get(status, status), detail))
        self.status = status


def lib():
    """Load the CUDA library (fails loudly when it has not been built: there is no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("liballegro_b200.so not built: run `python -m paper_2504_16068_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _check(status):
    if status != 0:
        raise AllegroError(status, lib().allegro_last_error().decode())


def _ptr(t):
    if t is None:
        return None
    assert t.is_contiguous(), "tensors handed to the library must be contiguous"
    return t.data_ptr()


def _stream(stream):
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


def torch_dtype(dtype):
    return torch.float32 if dtype == F32 else torch.float64


class Plan:
    """allegro_plan_t: CG table + path plan for (l_max, full parity), n channels, dtype, weight mode."""

    def __init__(self, l_max, n, dtype=F32, wmode=W_SCALAR):
        h = _vp()
        _check(lib().allegro_plan_create(l_max, 0, n, dtype, wmode, C.byref(h)))
        self.h = h
        self.l_max, self.n, self.dtype, self.wmode = l_max, n, dtype, wmode
        self.P = lib().allegro_plan_num_paths(h)
        self.dV = lib().allegro_plan_dim_v(h)
        self.dE = lib().allegro_plan_dim_e(h)
        self.nnz = lib().allegro_plan_nnz(h)
        self.tdtype = torch_dtype(dtype)

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.allegro_plan_destroy(self.h)
            self.h = None

    def bind_weights(self, path_w, stream=None):
        """scalar mode: fold path_w into the plan's combined tensor; later calls may pass path_w=None (CUDA-graph capturable)"""
        _check(lib().allegro_plan_bind_weights(self.h, _ptr(path_w), _stream(stream)))

    def set_out_blocks(self, block_mask):
        """compute only the output blocks of block_mask (bit b = block b in component order 0e, 0o, 1e, ...)"""
        _check(lib().allegro_plan_set_out_blocks(self.h, int(block_mask)))

    def set_in_blocks(self, block_mask):
        """input blocks of V that are present (same bit order); the others are taken as zero and never read"""
        _check(lib().allegro_plan_set_in_blocks(self.h, int(block_mask)))

    def paths(self):
        names = ["l1", "p1", "l2", "l3", "p3", "off1", "off2", "off3"]
        arrs = [np.zeros(self.P, dtype=np.int32) for _ in names]
        _check(lib().allegro_plan_paths(self.h, *[a.ctypes.data_as(_i32p) for a in arrs]))
        return dict(zip(names, arrs))

    def cg(self):
        path, i, j, k = [np.zeros(self.nnz, dtype=np.int32) for _ in range(4)]
        coef = np.zeros(self.nnz)
        _check(lib().allegro_plan_cg(self.h, *[a.ctypes.data_as(_i32p) for a in (path, i, j, k)], coef.ctypes.data_as(_f64p)))
        return dict(path=path, i=i, j=j, k=k, coef=coef)


def cg_real_block(l1, l2, l3):
    out = np.zeros((2 * l1 + 1, 2 * l2 + 1, 2 * l3 + 1))
    _check(lib().allegro_cg_real_block(l1, l2, l3, out.ctypes.data_as(_f64p)))
    return out


def segments_build(row_ptr_host, tile_edges):
    """HOST int32 row_ptr -> HOST int32 items[n_items, 3] (reading A16)."""
    rp = np.ascontiguousarray(row_ptr_host, dtype=np.int32)
    n_atoms = rp.shape[0] - 1
    cnt = C.c_long(0)
    _check(lib().allegro_segments_build(rp.ctypes.data_as(_i32p), n_atoms, tile_edges, None, 0, C.byref(cnt)))
    items = np.zeros((cnt.value, 3), dtype=np.int32)
    _check(lib().allegro_segments_build(rp.ctypes.data_as(_i32p), n_atoms, tile_edges, items.ctypes.data_as(_i32p), cnt.value,
                                        C.byref(cnt)))
    return items


def launch_count():
    return lib().allegro_launch_count()


def _n_items(items):
    return 0 if items is None else items.shape[0]


def env_workspace(plan, n_atoms, items):
    return lib().allegro_env_workspace(plan.h, n_atoms, _n_items(items))


def tp_backward_workspace(plan, n_atoms, n_edges, items, want_g_path_w):
    return lib().allegro_tp_backward_workspace(plan.h, n_atoms, n_edges, _n_items(items), int(bool(want_g_path_w)))


def _ws(nbytes, device):
    return torch.empty(max(int(nbytes), 16), dtype=torch.uint8, device=device)


def env_embed(plan, row_ptr, rvec, w, scale=1.0, items=None, Eenv=None, workspace=None, stream=None):
    n_atoms, n_edges = row_ptr.shape[0] - 1, rvec.shape[0]
    if Eenv is None:
        Eenv = torch.empty((n_atoms, plan.n, plan.dE), dtype=plan.tdtype, device=rvec.device)
    if workspace is None and items is not None:
        workspace = _ws(env_workspace(plan, n_atoms, items), rvec.device)
    _check(lib().allegro_env_embed(plan.h, n_atoms, n_edges, _ptr(row_ptr), _ptr(items), _n_items(items), _ptr(rvec), _ptr(w),
                                   float(scale), _ptr(Eenv), _ptr(workspace), 0 if workspace is None else workspace.numel(),
                                   _stream(stream)))
    return Eenv


def tp_forward(plan, row_ptr, V, Eenv, path_w, items=None, out=None, stream=None):
    n_atoms, n_edges = row_ptr.shape[0] - 1, V.shape[0]
    if out is None:
        out = torch.empty_like(V)
    _check(lib().allegro_tp_forward(plan.h, n_atoms, n_edges, _ptr(row_ptr), _ptr(items), _n_items(items), _ptr(V), _ptr(Eenv),
                                    _ptr(path_w), _ptr(out), _stream(stream)))
    return out


def tp_forward_aux(plan, row_ptr, V, Eenv, path_w, out, out_scalars, items=None, stream=None):
    """dense tp_forward that also writes the compact 0e scalars out_scalars[e][n] = out[e][n][0]"""
    n_atoms, n_edges = row_ptr.shape[0] - 1, V.shape[0]
    _check(lib().allegro_tp_forward_aux(plan.h, n_atoms, n_edges, _ptr(row_ptr), _ptr(items), _n_items(items), _ptr(V), _ptr(Eenv), _ptr(path_w),
                                        _ptr(out), _ptr(out_scalars), _stream(stream)))
    return out, out_scalars


def tp_backward_aux(plan, row_ptr, G, g_scalars, V, Eenv, path_w, gV, gEenv, items=None, workspace=None, stream=None):
    """dense tp_backward with the cotangent G + g_scalars (x) delta_0e (g_scalars [E, n] compact, may be None)"""
    n_atoms, n_edges = row_ptr.shape[0] - 1, V.shape[0]
    if workspace is None:
        workspace = _ws(tp_backward_workspace(plan, n_atoms, n_edges, items, False), V.device)
    _check(lib().allegro_tp_backward_aux(plan.h, n_atoms, n_edges, _ptr(row_ptr), _ptr(items), _n_items(items), _ptr(G), _ptr(g_scalars), _ptr(V),
                                         _ptr(Eenv), _ptr(path_w), _ptr(gV), _ptr(gEenv), _ptr(workspace), workspace.numel(), _stream(stream)))
    return gV, gEenv


def tp_forward_outer(plan, row_ptr, rvec, v0, Eenv, path_w, out, out_scalars=None, items=None, stream=None):
    """dense tp_forward whose input V0 = v0 (x) Y(rhat) is generated on chip (layer-1 specialisation)"""
    n_atoms, n_edges = row_ptr.shape[0] - 1, rvec.shape[0]
    _check(lib().allegro_tp_forward_outer(plan.h, n_atoms, n_edges, _ptr(row_ptr), _ptr(items), _n_items(items), _ptr(rvec), _ptr(v0), _ptr(Eenv),
                                          _ptr(path_w), _ptr(out), _ptr(out_scalars), _stream(stream)))
    return out, out_scalars


def tp_backward_outer(plan, row_ptr, G, g_scalars, rvec, v0, Eenv, path_w, g_v0, gY, gEenv, items=None, workspace=None, stream=None):
    """VJP of tp_forward_outer: g_v0 [E, n], gY [E, dE] (the contractions of gV0 with Y and with v0), gEenv"""
    n_atoms, n_edges = row_ptr.shape[0] - 1, rvec.shape[0]
    if workspace is None:
        workspace = _ws(tp_backward_workspace(plan, n_atoms, n_edges, items, False), rvec.device)
    _check(lib().allegro_tp_backward_outer(plan.h, n_atoms, n_edges, _ptr(row_ptr), _ptr(items), _n_items(items), _ptr(G), _ptr(g_scalars), _ptr(rvec),
                                           _ptr(v0), _ptr(Eenv), _ptr(path_w), _ptr(g_v0), _ptr(gY), _ptr(gEenv), _ptr(workspace), workspace.numel(),
                                           _stream(stream)))
    return g_v0, gY, gEenv


def edge_embed_factors(plan, rvec, W_x0, W_v0, r_cut, x0, v0, stream=None):
    _check(lib().allegro_edge_embed_factors(plan.h, rvec.shape[0], _ptr(rvec), _ptr(W_x0), _ptr(W_v0), W_x0.shape[1], float(r_cut), _ptr(x0), _ptr(v0),
                                            _stream(stream)))
    return x0, v0


def edge_embed_factors_backward(plan, rvec, W_x0, W_v0, r_cut, g_x0, g_v0, gY, g_rvec, stream=None):
    """g_rvec is accumulated into"""
    _check(lib().allegro_edge_embed_factors_backward(plan.h, rvec.shape[0], _ptr(rvec), _ptr(W_x0), _ptr(W_v0), W_x0.shape[1], float(r_cut), _ptr(g_x0),
                                                     _ptr(g_v0), _ptr(gY), _ptr(g_rvec), _stream(stream)))
    return g_rvec


def tp_forward_energy(plan, row_ptr, V, Eenv, path_w, q, kappa, items=None, want_out=True, want_e=True, want_G=True, out=None, e_edge=None,
                      G=None, stream=None):
    """-> (out or None, e_edge or None, G or None): tp_forward with the energy / cotangent epilogue fused"""
    n_atoms, n_edges = row_ptr.shape[0] - 1, V.shape[0]
    if out is None and want_out:
        out = torch.empty_like(V)
    if e_edge is None and want_e:
        e_edge = torch.empty((n_edges,), dtype=V.dtype, device=V.device)
    if G is None and want_G:
        G = torch.empty_like(V)
    _check(lib().allegro_tp_forward_energy(plan.h, n_atoms, n_edges, _ptr(row_ptr), _ptr(items), _n_items(items), _ptr(V), _ptr(Eenv),
                                           _ptr(path_w), _ptr(q), float(kappa), _ptr(out), _ptr(e_edge), _ptr(G), _stream(stream)))
    return out, e_edge, G


def tp_backward(plan, row_ptr, G, V, Eenv, path_w, items=None, want_gV=True, want_g_path_w=False, gV=None, gEenv=None,
                g_path_w=None, workspace=None, stream=None):
    """-> (gV or None, gEenv, g_path_w or None)"""
    n_atoms, n_edges = row_ptr.shape[0] - 1, V.shape[0]
    if gV is None and want_gV:
        gV = torch.empty_like(V)
    if gEenv is None:
        gEenv = torch.empty_like(Eenv)
    if g_path_w is None and want_g_path_w:
        g_path_w = torch.empty_like(path_w)
    if workspace is None:
        workspace = _ws(tp_backward_workspace(plan, n_atoms, n_edges, items, g_path_w is not None), V.device)
    _check(lib().allegro_tp_backward(plan.h, n_atoms, n_edges, _ptr(row_ptr), _ptr(items), _n_items(items), _ptr(G), _ptr(V),
                                     _ptr(Eenv), _ptr(path_w), _ptr(gV), _ptr(gEenv), _ptr(g_path_w), _ptr(workspace),
                                     workspace.numel(), _stream(stream)))
    return gV, gEenv, g_path_w


def tp_backward_static(plan, row_ptr, G, V, Eenv, path_w, gV, gEenv, g_path_w=None, items=None, stream=None):
    """allegro_tp_backward_static: the VJP with its scratch in the library's static device array -- no allocation anywhere, so
    every output tensor is the caller's (gV may be None).  -> (gV, gEenv, g_path_w)"""
    n_atoms, n_edges = row_ptr.shape[0] - 1, V.shape[0]
    _check(lib().allegro_tp_backward_static(plan.h, n_atoms, n_edges, _ptr(row_ptr), _ptr(items), _n_items(items), _ptr(G), _ptr(V), _ptr(Eenv),
                                            _ptr(path_w), _ptr(gV), _ptr(gEenv), _ptr(g_path_w), _stream(stream)))
    return gV, gEenv, g_path_w


def tp_backward_energy(plan, row_ptr, out, V, Eenv, path_w, q, kappa, items=None, want_gV=True, want_g_path_w=False, gV=None, gEenv=None,
                       g_path_w=None, workspace=None, stream=None):
    """-> (gV or None, gEenv, g_path_w or None); the cotangent G = q (x) delta + kappa out is formed in registers"""
    n_atoms, n_edges = row_ptr.shape[0] - 1, V.shape[0]
    if gV is None and want_gV:
        gV = torch.empty_like(V)
    if gEenv is None:
        gEenv = torch.empty_like(Eenv)
    if g_path_w is None and want_g_path_w:
        g_path_w = torch.empty_like(path_w)
    if workspace is None:
        workspace = _ws(tp_backward_workspace(plan, n_atoms, n_edges, items, g_path_w is not None), V.device)
    _check(lib().allegro_tp_backward_energy(plan.h, n_atoms, n_edges, _ptr(row_ptr), _ptr(items), _n_items(items), _ptr(out), _ptr(V),
                                            _ptr(Eenv), _ptr(path_w), _ptr(q), float(kappa), _ptr(gV), _ptr(gEenv), _ptr(g_path_w),
                                            _ptr(workspace), workspace.numel(), _stream(stream)))
    return gV, gEenv, g_path_w


def tp_fused_energy(plan, row_ptr, V, Eenv, path_w, q, kappa, items=None, want_gV=True, want_g_path_w=False, e_edge=None, gV=None, gEenv=None,
                    g_path_w=None, workspace=None, stream=None):
    """forward + energy + VJP in one kernel -> (e_edge, gV or None, gEenv, g_path_w or None); `out` never exists"""
    n_atoms, n_edges = row_ptr.shape[0] - 1, V.shape[0]
    if e_edge is None:
        e_edge = torch.empty((n_edges,), dtype=V.dtype, device=V.device)
    if gV is None and want_gV:
        gV = torch.empty_like(V)
    if gEenv is None:
        gEenv = torch.empty_like(Eenv)
    if g_path_w is None and want_g_path_w:
        g_path_w = torch.empty((plan.P,), dtype=V.dtype, device=V.device)
    if workspace is None:
        workspace = _ws(tp_backward_workspace(plan, n_atoms, n_edges, items, g_path_w is not None), V.device)
    _check(lib().allegro_tp_fused_energy(plan.h, n_atoms, n_edges, _ptr(row_ptr), _ptr(items), _n_items(items), _ptr(V), _ptr(Eenv), _ptr(path_w),
                                         _ptr(q), float(kappa), _ptr(e_edge), _ptr(gV), _ptr(gEenv), _ptr(g_path_w), _ptr(workspace),
                                         workspace.numel(), _stream(stream)))
    return e_edge, gV, gEenv, g_path_w


def tp_double_backward(plan, row_ptr, G, V, Eenv, path_w, aV, bE, want_d_path_w=True, stream=None):
    """second derivative (training): gradients of <aV, gV> + <bE, gEenv> -> (dG, dV, dEenv, d_path_w or None)"""
    n_atoms, n_edges = row_ptr.shape[0] - 1, V.shape[0]
    dG, dV, dE = torch.empty_like(V), torch.empty_like(V), torch.empty_like(Eenv)
    dw = torch.empty((plan.P,), dtype=V.dtype, device=V.device) if want_d_path_w else None
    ws = _ws(lib().allegro_tp_double_backward_workspace(plan.h, n_atoms, n_edges), V.device)
    _check(lib().allegro_tp_double_backward(plan.h, n_atoms, n_edges, _ptr(row_ptr), _ptr(G), _ptr(V), _ptr(Eenv), _ptr(path_w), _ptr(aV), _ptr(bE),
                                            _ptr(dG), _ptr(dV), _ptr(dE), _ptr(dw), _ptr(ws), ws.numel(), _stream(stream)))
    return dG, dV, dE, dw


def env_embed_backward(plan, row_ptr, gEenv, rvec, w, scale=1.0, want_g_w=True, g_rvec=None, g_w=None, stream=None):
    """-> (g_rvec[E,3], g_w[E,n] or None)"""
    n_atoms, n_edges = row_ptr.shape[0] - 1, rvec.shape[0]
    if g_rvec is None:
        g_rvec = torch.empty_like(rvec)
    if g_w is None and want_g_w:
        g_w = torch.empty_like(w)
    _check(lib().allegro_env_embed_backward(plan.h, n_atoms, n_edges, _ptr(row_ptr), _ptr(gEenv), _ptr(rvec), _ptr(w),
                                            float(scale), _ptr(g_rvec), _ptr(g_w), _stream(stream)))
    return g_rvec, g_w


def _dt(t):
    return F32 if t.dtype == torch.float32 else F64


def force_gather(row_ptr, rev, g_rvec, F=None, stream=None):
    n_atoms, n_edges = row_ptr.shape[0] - 1, g_rvec.shape[0]
    if F is None:
        F = torch.empty((n_atoms, 3), dtype=g_rvec.dtype, device=g_rvec.device)
    _check(lib().allegro_force_gather(n_atoms, n_edges, _ptr(row_ptr), _ptr(rev), _ptr(g_rvec), _dt(g_rvec), _ptr(F), _stream(stream)))
    return F


def radial_forward(rvec, W_r, r_cut, w=None, stream=None):
    n, nb = W_r.shape
    if w is None:
        w = torch.empty((rvec.shape[0], n), dtype=rvec.dtype, device=rvec.device)
    _check(lib().allegro_radial_forward(n, nb, float(r_cut), _dt(rvec), rvec.shape[0], _ptr(rvec), _ptr(W_r), _ptr(w), _stream(stream)))
    return w


def radial_backward(rvec, W_r, r_cut, g_w, g_rvec, stream=None):
    """g_rvec += (sum_n g_w dw/dr) rhat, in place"""
    n, nb = W_r.shape
    _check(lib().allegro_radial_backward(n, nb, float(r_cut), _dt(rvec), rvec.shape[0], _ptr(rvec), _ptr(W_r), _ptr(g_w), _ptr(g_rvec),
                                         _stream(stream)))
    return g_rvec


def env_radial_forward(plan, row_ptr, rvec, W_r, r_cut, scale=1.0, items=None, want_w=False, w=None, Eenv=None, workspace=None, stream=None):
    """-> (Eenv, w or None): radial weights + Y_lm + environment embedding in one kernel"""
    n_atoms, n_edges = row_ptr.shape[0] - 1, rvec.shape[0]
    if Eenv is None:
        Eenv = torch.empty((n_atoms, plan.n, plan.dE), dtype=plan.tdtype, device=rvec.device)
    if w is None and want_w:
        w = torch.empty((n_edges, plan.n), dtype=plan.tdtype, device=rvec.device)
    if workspace is None and items is not None:
        workspace = _ws(env_workspace(plan, n_atoms, items), rvec.device)
    _check(lib().allegro_env_radial_forward(plan.h, n_atoms, n_edges, _ptr(row_ptr), _ptr(items), _n_items(items), _ptr(rvec), _ptr(W_r),
                                            W_r.shape[1], float(r_cut), float(scale), _ptr(w), _ptr(Eenv), _ptr(workspace),
                                            0 if workspace is None else workspace.numel(), _stream(stream)))
    return Eenv, w


def env_radial_backward(plan, row_ptr, gEenv, rvec, W_r, r_cut, scale=1.0, want_g_w=False, g_rvec=None, g_w=None, stream=None):
    """-> (g_rvec[E,3] complete dE/dr_e, g_w or None): embedding VJP + radial chain rule in one kernel"""
    n_atoms, n_edges = row_ptr.shape[0] - 1, rvec.shape[0]
    if g_rvec is None:
        g_rvec = torch.empty_like(rvec)
    if g_w is None and want_g_w:
        g_w = torch.empty((n_edges, plan.n), dtype=plan.tdtype, device=rvec.device)
    _check(lib().allegro_env_radial_backward(plan.h, n_atoms, n_edges, _ptr(row_ptr), _ptr(gEenv), _ptr(rvec), _ptr(W_r), W_r.shape[1],
                                             float(r_cut), float(scale), _ptr(g_rvec), _ptr(g_w), _stream(stream)))
    return g_rvec, g_w


def edge_energy(plan, out, q, kappa, want_e=True, want_G=True, e_edge=None, G=None, stream=None):
    """-> (e_edge[E] or None, G or None)"""
    if e_edge is None and want_e:
        e_edge = torch.empty((out.shape[0],), dtype=out.dtype, device=out.device)
    if G is None and want_G:
        G = torch.empty_like(out)
    _check(lib().allegro_edge_energy(plan.h, out.shape[0], _ptr(out), _ptr(q), float(kappa), _ptr(e_edge), _ptr(G), _stream(stream)))
    return e_edge, G


def virial(rvec, g_rvec, W=None, stream=None):
    """-> W [3,3]: W[a][b] = sum_e g_rvec[e][a] rvec[e][b]"""
    if W is None:
        W = torch.empty((3, 3), dtype=rvec.dtype, device=rvec.device)
    _check(lib().allegro_virial(rvec.shape[0], _ptr(rvec), _ptr(g_rvec), _dt(rvec), _ptr(W), _stream(stream)))
    return W


def check_graph(row_ptr, n_edges, items=None, rev=None, col=None, rvec=None, stream=None):
    """debugging aid (allegro_check_graph): number of violations in the step's index lists; raises AllegroError when there is one"""
    n_bad = C.c_long(-1)
    dt = _dt(rvec) if rvec is not None else F32
    n_items = 0 if items is None else items.numel() // 3
    _check(lib().allegro_check_graph(row_ptr.shape[0] - 1, int(n_edges), _ptr(row_ptr), _ptr(items), n_items, _ptr(rev), _ptr(col), _ptr(rvec), dt,
                                     C.byref(n_bad), _stream(stream)))
    return n_bad.value


def segment_sum(ptr, vals, out=None, stream=None):
    nseg = ptr.shape[0] - 1
    if out is None:
        out = torch.empty((nseg,), dtype=vals.dtype, device=vals.device)
    _check(lib().allegro_segment_sum(_ptr(ptr), nseg, _ptr(vals), _dt(vals), _ptr(out), _stream(stream)))
    return out


# ---------------------------------------------------------------------------------------------------- two-layer model helpers
def edge_embed(plan, rvec, W_x0, W_v0, r_cut, x0=None, V0=None, stream=None):
    E = rvec.shape[0]
    if x0 is None:
        x0 = torch.empty((E, plan.n), dtype=plan.tdtype, device=rvec.device)
    if V0 is None:
        V0 = torch.empty((E, plan.n, plan.dV), dtype=plan.tdtype, device=rvec.device)
    _check(lib().allegro_edge_embed(plan.h, E, _ptr(rvec), _ptr(W_x0), _ptr(W_v0), W_x0.shape[1], float(r_cut), _ptr(x0), _ptr(V0), _stream(stream)))
    return x0, V0


def edge_embed_backward(plan, rvec, W_x0, W_v0, r_cut, g_x0, gV0, g_rvec, stream=None):
    """g_rvec += ..., in place"""
    _check(lib().allegro_edge_embed_backward(plan.h, rvec.shape[0], _ptr(rvec), _ptr(W_x0), _ptr(W_v0), W_x0.shape[1], float(r_cut), _ptr(g_x0),
                                             _ptr(gV0), _ptr(g_rvec), _stream(stream)))
    return g_rvec


def linear(x, W, transpose_w=False, y=None, accumulate=False, stream=None):
    """y (+)= x W^T (transpose_w False, W [n_out, n_in]) or x W (transpose_w True, W [n_in, n_out])"""
    n_in = x.shape[1]
    n_out = W.shape[1] if transpose_w else W.shape[0]
    if y is None:
        assert not accumulate
        y = torch.empty((x.shape[0], n_out), dtype=x.dtype, device=x.device)
    _check(lib().allegro_linear(x.shape[0], n_out, n_in, _dt(x), _ptr(x), _ptr(W), int(transpose_w), int(accumulate), _ptr(y), _stream(stream)))
    return y


def latent_forward(rvec, r_cut, x, V, A, z=None, x_new=None, stream=None):
    """-> (z, x_new)"""
    if z is None:
        z = torch.empty_like(x)
    if x_new is None:
        x_new = torch.empty_like(x)
    _check(lib().allegro_latent_forward(x.shape[0], x.shape[1], V.shape[2], float(r_cut), _dt(x), _ptr(rvec), _ptr(x), _ptr(V), _ptr(A), _ptr(z),
                                        _ptr(x_new), _stream(stream)))
    return z, x_new


def latent_backward(rvec, r_cut, z, g_xnew, A, gV, g_rvec, g_x=None, stream=None):
    """-> g_x (overwritten); gV[:, :, 0] and g_rvec are accumulated into"""
    if g_x is None:
        g_x = torch.empty_like(z)
    _check(lib().allegro_latent_backward(z.shape[0], z.shape[1], gV.shape[2], float(r_cut), _dt(z), _ptr(rvec), _ptr(z), _ptr(g_xnew), _ptr(A),
                                         _ptr(g_x), _ptr(gV), _ptr(g_rvec), _stream(stream)))
    return g_x


def add_inplace(y, x, stream=None):
    _check(lib().allegro_add_inplace(y.numel(), _dt(y), _ptr(y), _ptr(x), _stream(stream)))
    return y


class LayerStepGraph:
    """allegro_step_t: the single-layer MD step for device-resident buffers, captured into a CUDA graph INSIDE the library and
    replayed with one launch.  `plan` must have its weights bound; F [N,3] and e_tot [1] are written by every launch."""

    def __init__(self, plan, row_ptr, rev, rvec, V, W_r, r_cut, q, kappa, scale, F, e_tot, want_gV=True):
        self.plan = plan
        self.N, self.E = row_ptr.shape[0] - 1, rvec.shape[0]
        self.refs = (row_ptr, rev, rvec, V, W_r, q, F, e_tot)          # the graph holds their addresses
        nbytes = lib().allegro_layer_step_workspace(plan.h, self.N, self.E, int(bool(want_gV)))
        self.ws = torch.empty(max(nbytes, 16), dtype=torch.uint8, device=rvec.device)
        h = _vp()
        _check(lib().allegro_layer_step_create(plan.h, self.N, self.E, _ptr(row_ptr), _ptr(rev), _ptr(rvec), _ptr(V), _ptr(W_r), W_r.shape[1],
                                               float(r_cut), _ptr(q), float(kappa), float(scale), int(bool(want_gV)), _ptr(F), _ptr(e_tot),
                                               _ptr(self.ws), self.ws.numel(), C.byref(h)))
        self.h = h
        self.F, self.e_tot = F, e_tot
        self.kernels_per_step = lib().allegro_layer_step_num_kernels(h)

    def buffer(self, name, shape, dtype):
        """view of a workspace buffer ("Eenv", "gEenv", "out", "gV", "e_edge", "g_rvec") as a tensor"""
        p = lib().allegro_layer_step_buffer(self.h, name.encode())
        if not p:
            return None
        off = p - self.ws.data_ptr()
        n = int(np.prod(shape)) * torch.empty((), dtype=dtype).element_size()
        return self.ws[off:off + n].view(dtype).view(*shape)

    def run(self, stream=None, mark=False):
        _check(lib().allegro_layer_step_launch(self.h, _stream(stream)))
        return self.F, self.e_tot

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.allegro_layer_step_destroy(self.h)
            self.h = None


def neighbour_list(pos, r_cut, box=None, mol_id=None, dtype=F32, species=None, rc_table=None, stream=None):
    """positions (device, float64 [N,3]) -> dict(row_ptr, col, rev, rvec[, rc_edge]) on the device (allegro_neighbour_count / _fill).
    box: cubic periodic box edge, or None for an open system (the bounding box is taken from the positions).
    species (int32 [N]) + rc_table (float64 [S,S], symmetric, <= r_cut): per-edge-type cutoffs; rc_edge [E] is returned as well."""
    assert pos.dtype == torch.float64 and pos.is_cuda
    N = pos.shape[0]
    ws = torch.empty(max(lib().allegro_neighbour_workspace(N), 16), dtype=torch.uint8, device=pos.device)
    row_ptr = torch.empty((N + 1,), dtype=torch.int32, device=pos.device)
    lo = hi = None
    if box is None:
        lo = np.ascontiguousarray(pos.min(0).values.cpu().numpy() if N else np.zeros(3))
        hi = np.ascontiguousarray(pos.max(0).values.cpu().numpy() if N else np.ones(3))
    plo = None if lo is None else lo.ctypes.data_as(_f64p)
    phi = None if hi is None else hi.ctypes.data_as(_f64p)
    n_edges = C.c_long(0)
    b = float(box) if box is not None else 0.0
    typed = species is not None and rc_table is not None
    ns = int(rc_table.shape[0]) if typed else 0
    _check(lib().allegro_neighbour_count(N, _ptr(pos), b, plo, phi, float(r_cut), _ptr(mol_id), _ptr(species) if typed else None, ns,
                                         _ptr(rc_table) if typed else None, _ptr(row_ptr), _ptr(ws), ws.numel(), _stream(stream), C.byref(n_edges)))
    E = n_edges.value
    col = torch.empty((E,), dtype=torch.int32, device=pos.device)
    rev = torch.empty((E,), dtype=torch.int32, device=pos.device)
    rvec = torch.empty((E, 3), dtype=torch_dtype(dtype), device=pos.device)
    rc_edge = torch.empty((E,), dtype=torch_dtype(dtype), device=pos.device) if typed else None
    _check(lib().allegro_neighbour_fill(N, _ptr(pos), b, plo, phi, float(r_cut), _ptr(mol_id), _ptr(species) if typed else None, ns,
                                        _ptr(rc_table) if typed else None, _ptr(row_ptr), E, _ptr(col), _ptr(rev), _ptr(rvec), _ptr(rc_edge),
                                        dtype, _ptr(ws), ws.numel(), _stream(stream)))
    out = dict(row_ptr=row_ptr, col=col, rev=rev, rvec=rvec)
    if typed:
        out["rc_edge"] = rc_edge
    return out


def env_linear_forward(plan, row_ptr, rvec, x, W, scale=1.0, Eenv=None, stream=None):
    """Eenv of the linear per-edge weights w = x W^T without forming w (allegro_env_linear_forward)"""
    n_atoms = row_ptr.shape[0] - 1
    if Eenv is None:
        Eenv = torch.empty((n_atoms, plan.n, plan.dE), dtype=rvec.dtype, device=rvec.device)
    _check(lib().allegro_env_linear_forward(plan.h, n_atoms, rvec.shape[0], _ptr(row_ptr), _ptr(rvec), _ptr(x), _ptr(W), x.shape[1], float(scale),
                                            _ptr(Eenv), _stream(stream)))
    return Eenv


def env_linear_backward(plan, row_ptr, gEenv, rvec, x, W, scale, g_rvec, g_x, accumulate_g_rvec=False, accumulate_g_x=False, stream=None):
    """VJP of env_linear_forward: g_rvec [E,3] and g_x [E,n_in] are overwritten or accumulated into"""
    n_atoms = row_ptr.shape[0] - 1
    _check(lib().allegro_env_linear_backward(plan.h, n_atoms, rvec.shape[0], _ptr(row_ptr), _ptr(gEenv), _ptr(rvec), _ptr(x), _ptr(W), x.shape[1],
                                             float(scale), _ptr(g_rvec), int(bool(accumulate_g_rvec)), _ptr(g_x), int(bool(accumulate_g_x)),
                                             _stream(stream)))
    return g_rvec, g_x


def env_radial_forward_typed(plan, row_ptr, rvec, W_r, rc_edge, scale=1.0, items=None, want_w=False, w=None, Eenv=None, workspace=None, stream=None):
    """env_radial_forward with a cutoff radius per edge (per-edge-type cutoffs, reading A27) -> (Eenv, w or None)"""
    n_atoms, n_edges = row_ptr.shape[0] - 1, rvec.shape[0]
    if Eenv is None:
        Eenv = torch.empty((n_atoms, plan.n, plan.dE), dtype=rvec.dtype, device=rvec.device)
    if w is None and want_w:
        w = torch.empty((n_edges, plan.n), dtype=rvec.dtype, device=rvec.device)
    if workspace is None:
        workspace = _ws(env_workspace(plan, n_atoms, items), rvec.device)
    _check(lib().allegro_env_radial_forward_typed(plan.h, n_atoms, n_edges, _ptr(row_ptr), _ptr(items), _n_items(items), _ptr(rvec), _ptr(W_r),
                                                  W_r.shape[1], _ptr(rc_edge), float(scale), _ptr(w), _ptr(Eenv), _ptr(workspace), workspace.numel(),
                                                  _stream(stream)))
    return Eenv, w


def env_radial_backward_typed(plan, row_ptr, gEenv, rvec, W_r, rc_edge, scale=1.0, want_g_w=False, g_rvec=None, g_w=None, stream=None):
    """VJP of env_radial_forward_typed -> (g_rvec, g_w or None)"""
    n_atoms, n_edges = row_ptr.shape[0] - 1, rvec.shape[0]
    if g_rvec is None:
        g_rvec = torch.empty_like(rvec)
    if g_w is None and want_g_w:
        g_w = torch.empty((n_edges, plan.n), dtype=rvec.dtype, device=rvec.device)
    _check(lib().allegro_env_radial_backward_typed(plan.h, n_atoms, n_edges, _ptr(row_ptr), _ptr(gEenv), _ptr(rvec), _ptr(W_r), W_r.shape[1],
                                                   _ptr(rc_edge), float(scale), _ptr(g_rvec), _ptr(g_w), _stream(stream)))
    return g_rvec, g_w


def measure_peaks(stream=None):
    """-> dict(fp32_fma_tflops, tf32_mma_tflops): roofline denominators measured on the current device"""
    a, b = C.c_double(0.0), C.c_double(0.0)
    _check(lib().allegro_measure_fp32_fma_peak(_stream(stream), C.byref(a)))
    _check(lib().allegro_measure_tf32_mma_peak(_stream(stream), C.byref(b)))
    by_n = {}
    for n in (32, 80, 128, 256):
        c = C.c_double(0.0)
        _check(lib().allegro_measure_tf32_mma_rate(n, _stream(stream), C.byref(c)))
        by_n[str(n)] = c.value
    return dict(fp32_fma_tflops=a.value, tf32_mma_tflops=b.value, tf32_mma_tflops_by_N=by_n)


def layer_step_host_workspace(plan, n_atoms, n_edges, n_basis, want_gV=True):
    return lib().allegro_layer_step_host_workspace(plan.h, n_atoms, n_edges, n_basis, int(bool(want_gV)))


def layer_step_host(plan, row_ptr, rev, rvec, V, W_r, r_cut, path_w, q, kappa, scale, F, e_tot, workspace, want_gV=True, stream=None):
    """All tensor arguments except `workspace` are HOST tensors (ideally pinned); F [N,3] and e_tot [1] are filled on return."""
    for t in (row_ptr, rev, rvec, V, W_r, path_w, q, F, e_tot):
        assert not t.is_cuda and t.is_contiguous()
    _check(lib().allegro_layer_step_host(plan.h, row_ptr.shape[0] - 1, rvec.shape[0], _ptr(row_ptr), _ptr(rev), _ptr(rvec), _ptr(V), _ptr(W_r),
                                         W_r.shape[1], float(r_cut), _ptr(path_w), _ptr(q), float(kappa), float(scale), int(bool(want_gV)),
                                         _ptr(F), _ptr(e_tot), _ptr(workspace), workspace.numel(), _stream(stream)))
    return F, e_tot

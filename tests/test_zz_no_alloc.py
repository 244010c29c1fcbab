"""allegro_tp_backward_static: the tensor-product VJP with its scratch in the library's file-scope device array (no cudaMalloc, no
caller workspace) against the existing allegro_tp_backward on the same inputs.  Collected last on purpose (file name): the
suite runs with pytest -x."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.join(ROOT, "tests")):
    if p not in sys.path:
        sys.path.insert(0, p)

import _chain  # noqa: E402

pytestmark = pytest.mark.gpu


def _rel(a, b):
    a, b = a.double(), b.double()
    den = float(b.abs().max())
    return float((a - b).abs().max()) / den if den > 0 else float((a - b).abs().max())


@pytest.mark.parametrize("name", ["C4s", "C0"])
def test_static_scratch_vjp_matches_workspace_path_twice(name):
    import torch

    import paper_2504_16068_b200 as ab
    from workloads import rng
    inp = _chain.make_inputs(name)
    dev = _chain.to_device(inp)
    dt = inp["dt"]
    tol = _chain.TOL[dt]
    plan = ab.Plan(inp["lmax"], inp["n"], ab.F64 if dt == np.float64 else ab.F32)
    rp, V, pw = dev["row_ptr"], dev["V"], dev["path_w"]
    N, E = inp["N"], inp["E"]
    Eenv = torch.from_numpy((rng.normal(31, rng.STREAMS["W_w"], (N, inp["n"], plan.dE)) * 0.5).astype(dt)).cuda()
    items = torch.from_numpy(ab.segments_build(inp["row_ptr"], 7)).cuda()
    assert ab.lib().allegro_tp_backward_static_capacity() == 4 << 20
    # two calls in a row with different cotangents (the array keeps the first call's contents), then with the centres split into items
    for rep, it in ((0, None), (1, None), (2, items)):
        G = torch.from_numpy(rng.normal(40 + rep, rng.STREAMS["G"], (E, inp["n"], plan.dV)).astype(dt)).cuda()
        gV_ref, gE_ref, gw_ref = ab.tp_backward(plan, rp, G, V, Eenv, pw, items=it, want_g_path_w=True)
        gV, gE, gw = torch.empty_like(V), torch.empty_like(Eenv), torch.empty_like(pw)
        ab.tp_backward_static(plan, rp, G, V, Eenv, pw, gV, gE, gw, items=it)
        torch.cuda.synchronize()
        for nm, a, b in (("gV", gV, gV_ref), ("gEenv", gE, gE_ref), ("g_path_w", gw, gw_ref)):
            assert _rel(a, b) <= tol, "%s call %d: %s differs by %g" % (name, rep, nm, _rel(a, b))


def test_static_scratch_rejects_what_does_not_fit():
    import torch

    import paper_2504_16068_b200 as ab
    plan = ab.Plan(2, 64, ab.F32)
    N = 200000                                   # 200,000 x 30 x 4 B = 24 MB of path-weight partial rows > 4 MiB
    rp = torch.zeros(N + 1, dtype=torch.int32, device="cuda")
    V = torch.zeros((0, 64, 18), device="cuda")
    Eenv = torch.zeros((N, 64, 9), device="cuda")
    pw = torch.ones(30, device="cuda")
    with pytest.raises(ab.AllegroError) as ei:
        ab.tp_backward_static(plan, rp, V, V, Eenv, pw, None, torch.empty_like(Eenv), torch.empty_like(pw))
    assert ei.value.status == 4 and "static array holds" in str(ei.value)
    dense = ab.Plan(2, 64, ab.F32, ab.W_DENSE)   # the dense path allocates: not served by this entry point
    with pytest.raises(ab.AllegroError) as ei:
        ab.tp_backward_static(dense, rp[:2], V, V, Eenv[:1], pw, None, torch.empty_like(Eenv[:1]), None)
    assert ei.value.status == 2

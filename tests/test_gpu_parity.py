"""GPU parity: the CUDA library (through the C ABI) against the float64 oracle, element by element, on the
same seeded inputs.  Tolerances are BASELINE.json:north_star's (reading A10): per tensor
max|d| <= 1e-5 max|ref| (fp32), 1e-11 (fp64); forces <= 1e-4 relative RMS (fp32); integers bit-exact."""
import numpy as np
import pytest

import _chain

pytestmark = pytest.mark.gpu

KEYS = ("w", "Eenv", "out", "e_edge", "G", "gV", "gEenv", "g_path_w", "g_w", "g_r_env", "g_r", "F", "E_mol")


def _assert_close(ref, got, dt, keys=KEYS, rows=None, label=""):
    errs = _chain.compare(ref, got, dt, keys, rows)
    tol = _chain.TOL[dt]
    bad = {k: v for k, v in errs.items() if not v <= tol}
    assert not bad, "%s: over tolerance %g: %s (all: %s)" % (label, tol, bad, errs)
    if "F" in errs and "F" in ref:
        F = got["F"].cpu().numpy().astype(np.float64)
        rms = np.linalg.norm(F - ref["F"]) / np.linalg.norm(ref["F"])
        assert rms <= _chain.FORCE_RMS_TOL[dt], "%s: force relative RMS %g" % (label, rms)
    return errs


# C0 is BASELINE.json:configs[0] in full; the *s variants are the other configs' recipes at sizes the oracle
# finishes in seconds (they still span many tiles and ragged tails: degrees are not multiples of the slot count)
@pytest.mark.parametrize("name", ["C0", "C1s", "C3s", "C4s"])
def test_chain_matches_oracle(name):
    inp = _chain.make_inputs(name)
    ref = _chain.oracle_chain(inp)
    got = _chain.gpu_chain(inp)
    errs = _assert_close(ref, got, inp["dt"], label=name)
    print(name, {k: "%.2e" % v for k, v in errs.items()})
    # sum of forces vanishes (Newton's third law: every edge has its reverse)
    F = got["F"].cpu().numpy().astype(np.float64)
    assert np.abs(F.sum(0)).max() <= 1e-3 * np.abs(F).max() * (1.0 if inp["dt"] == np.float32 else 1e-8)


@pytest.mark.parametrize("name", ["C0", "C1s", "C3s", "C4s"])
@pytest.mark.parametrize("want_out", [True, False])
def test_forward_energy_epilogue(name, want_out):
    """tp_forward_energy (out, e_edge, G from one kernel) against the oracle's tp_forward + edge_energy"""
    import oracle as orc
    import paper_2504_16068_b200 as ab
    inp = _chain.make_inputs(name)
    dev = _chain.to_device(inp)
    f8 = lambda a: np.asarray(a, dtype=np.float64)
    w, _ = orc.radial(f8(inp["W_r"]), inp["rc"], f8(inp["rvec"]))
    Eenv = orc.env_embed(inp["lmax"], inp["row_ptr"], f8(inp["rvec"]), w, inp["scale"])
    ref_out = orc.tp_forward(inp["lmax"], inp["row_ptr"], f8(inp["V"]), Eenv, f8(inp["path_w"]))
    ref_e, ref_G = orc.edge_energy(inp["lmax"], ref_out, f8(inp["q"]), inp["kappa"])
    plan = ab.Plan(inp["lmax"], inp["n"], ab.F64 if inp["dt"] == np.float64 else ab.F32)
    import torch
    Ed = torch.from_numpy(Eenv.astype(inp["dt"])).cuda()
    for items in (None, ab.segments_build(inp["row_ptr"], 7)):
        it = None if items is None else torch.from_numpy(items).cuda()
        out, e, G = ab.tp_forward_energy(plan, dev["row_ptr"], dev["V"], Ed, dev["path_w"], dev["q"], inp["kappa"], items=it, want_out=want_out)
        got = dict(out=out, e_edge=e, G=G)
        assert (out is None) == (not want_out)
        _assert_close(dict(out=ref_out, e_edge=ref_e, G=ref_G), got, inp["dt"], keys=("out", "e_edge", "G"), label=name)
    # e_edge only next to out (no G)
    out, e, G = ab.tp_forward_energy(plan, dev["row_ptr"], dev["V"], Ed, dev["path_w"], dev["q"], inp["kappa"], want_G=False)
    assert G is None
    _assert_close(dict(out=ref_out, e_edge=ref_e), dict(out=out, e_edge=e), inp["dt"], keys=("out", "e_edge"), label=name)


@pytest.mark.parametrize("name", ["C0", "C1s", "C3s", "C4s"])
@pytest.mark.parametrize("mode,fused_geometry", [("separate", False), ("epilogue", False), ("onthefly", False), ("onthefly", True), ("fused", True)])
def test_single_layer_step_modes(name, mode, fused_geometry):
    """the three call sequences of pipeline.SingleLayerStep (the object bench.py times) give the oracle's forces,
    energies and gradients; "onthefly" exercises tp_backward_energy (cotangent formed from out in registers)"""
    import torch

    import paper_2504_16068_b200 as ab
    from paper_2504_16068_b200.pipeline import SingleLayerStep
    inp = _chain.make_inputs(name)
    ref = _chain.oracle_chain(inp)
    dev = _chain.to_device(inp)
    plan = ab.Plan(inp["lmax"], inp["n"], ab.F64 if inp["dt"] == np.float64 else ab.F32)
    for items in (None, ab.segments_build(inp["row_ptr"], 9)):
        it = None if items is None else torch.from_numpy(items).cuda()
        st = SingleLayerStep(plan, dev, inp["rc"], inp["kappa"], inp["scale"], want_g_path_w=True, items=it, mode=mode, fused_geometry=fused_geometry)
        st.run()
        got = dict(w=st.w, Eenv=st.Eenv, out=st.out, e_edge=st.e_edge, G=st.G, gV=st.gV, gEenv=st.gEenv, g_path_w=st.g_path_w,
                   g_w=st.g_w, g_r=st.g_r, F=st.F)
        _assert_close(ref, got, inp["dt"], label="%s/%s" % (name, mode))
        e_ref = float(np.sum(ref["e_edge"]))
        assert abs(float(st.e_tot.item()) - e_ref) <= _chain.TOL[inp["dt"]] * max(abs(e_ref), float(np.abs(ref["e_edge"]).max()))
        # force-only VJP (gV = NULL) gives the same gEenv bits or values within tolerance
        st2 = SingleLayerStep(plan, dev, inp["rc"], inp["kappa"], inp["scale"], want_gV=False, items=it, mode=mode, fused_geometry=fused_geometry)
        st2.run()
        _assert_close(ref, dict(gEenv=st2.gEenv, F=st2.F), inp["dt"], keys=("gEenv", "F"), label="%s/%s/force-only" % (name, mode))


@pytest.mark.parametrize("name", ["C0", "C1s", "C3s", "C4s"])
def test_fused_geometry_kernels(name):
    """env_radial_forward / env_radial_backward with their optional outputs w, g_w against the oracle's
    radial + env_embed / env_embed_backward + radial_backward"""
    import oracle as orc
    import torch

    import paper_2504_16068_b200 as ab
    inp = _chain.make_inputs(name)
    dev = _chain.to_device(inp)
    ref = _chain.oracle_chain(inp)
    plan = ab.Plan(inp["lmax"], inp["n"], ab.F64 if inp["dt"] == np.float64 else ab.F32)
    for items in (None, ab.segments_build(inp["row_ptr"], 11)):
        it = None if items is None else torch.from_numpy(items).cuda()
        Eenv, w = ab.env_radial_forward(plan, dev["row_ptr"], dev["rvec"], dev["W_r"], inp["rc"], inp["scale"], items=it, want_w=True)
        _assert_close(ref, dict(Eenv=Eenv, w=w), inp["dt"], keys=("Eenv", "w"), label=name)
    gE = torch.from_numpy(ref["gEenv"].astype(inp["dt"])).cuda()
    g_r, g_w = ab.env_radial_backward(plan, dev["row_ptr"], gE, dev["rvec"], dev["W_r"], inp["rc"], inp["scale"], want_g_w=True)
    _assert_close(ref, dict(g_r=g_r, g_w=g_w), inp["dt"], keys=("g_r", "g_w"), label=name)
    g_r2, none = ab.env_radial_backward(plan, dev["row_ptr"], gE, dev["rvec"], dev["W_r"], inp["rc"], inp["scale"])
    assert none is None       # without g_w the factorised kernel runs (sums regrouped exactly): same values within tolerance
    _assert_close(ref, dict(g_r=g_r2), inp["dt"], keys=("g_r",), label=name + "/factorised")
    Eenv2, none = ab.env_radial_forward(plan, dev["row_ptr"], dev["rvec"], dev["W_r"], inp["rc"], inp["scale"])
    assert none is None
    _assert_close(ref, dict(Eenv=Eenv2), inp["dt"], keys=("Eenv",), label=name + "/factorised")
    it = torch.from_numpy(ab.segments_build(inp["row_ptr"], 11)).cuda()
    Eenv3, _ = ab.env_radial_forward(plan, dev["row_ptr"], dev["rvec"], dev["W_r"], inp["rc"], inp["scale"], items=it)
    _assert_close(ref, dict(Eenv=Eenv3), inp["dt"], keys=("Eenv",), label=name + "/factorised/items")


def test_c4_fp64_variant():
    """configs[4] asks for fp32 and fp64: the same molecule batch in double"""
    inp = _chain.make_inputs("C4s")
    for k in ("rvec", "V", "W_r", "path_w", "q"):
        inp[k] = inp[k].astype(np.float64)      # the fp32-rounded values, promoted: same numbers as the fp32 run
    inp["dt"] = np.float64
    ref = _chain.oracle_chain(inp)
    got = _chain.gpu_chain(inp)
    _assert_close(ref, got, np.float64, label="C4s/f64")


@pytest.mark.parametrize("name,T", [("C0", 5), ("C1s", 32), ("C4s", 7)])
def test_segment_items_split_centres(name, T):
    """A16: centres split over several items (tile_edges below the degree) give the same result as one item
    per centre; partial sums are combined in item order"""
    import oracle as orc
    import paper_2504_16068_b200 as ab
    inp = _chain.make_inputs(name)
    items = ab.segments_build(inp["row_ptr"], T)
    assert np.array_equal(items, orc.segments(inp["row_ptr"], T))          # integer plan: bit-exact
    assert items.shape[0] > inp["N"]
    ref = _chain.oracle_chain(inp)
    got = _chain.gpu_chain(inp, items=items)
    _assert_close(ref, got, inp["dt"], label="%s/T=%d" % (name, T))


def test_bitwise_determinism():
    """no float atomics anywhere: two runs give identical bits (reading A11)"""
    import torch
    inp = _chain.make_inputs("C1s")
    dev = _chain.to_device(inp)
    a = _chain.gpu_chain(inp, dev)
    b = _chain.gpu_chain(inp, dev)
    for k in a:
        if a[k] is not None:
            assert torch.equal(a[k], b[k]), k


def test_empty_and_degenerate_graphs():
    import torch

    import paper_2504_16068_b200 as ab
    plan = ab.Plan(2, 32, ab.F32)
    dev = "cuda"
    # (i) no atoms, no edges
    rp = torch.zeros(1, dtype=torch.int32, device=dev)
    z3 = torch.zeros((0, 3), device=dev)
    zV = torch.zeros((0, 32, 18), device=dev)
    zw = torch.zeros((0, 32), device=dev)
    pw = torch.ones(30, device=dev)
    E = ab.env_embed(plan, rp, z3, zw)
    assert E.shape == (0, 32, 9)
    out = ab.tp_forward(plan, rp, zV, E, pw)
    gV, gE, gpw = ab.tp_backward(plan, rp, zV, zV, E, pw, want_g_path_w=True)
    assert out.shape[0] == 0 and float(gpw.abs().sum()) == 0.0
    # (ii) atoms without neighbours (degree 0) between atoms with neighbours
    rp = torch.tensor([0, 0, 3, 3, 5, 5], dtype=torch.int32, device=dev)
    g = torch.Generator(device="cpu").manual_seed(1)
    rvec = torch.randn((5, 3), generator=g).to(dev)
    w = torch.randn((5, 32), generator=g).to(dev)
    V = torch.randn((5, 32, 18), generator=g).to(dev)
    E = ab.env_embed(plan, rp, rvec, w)
    assert float(E[0].abs().sum()) == 0.0 and float(E[2].abs().sum()) == 0.0 and float(E[4].abs().sum()) == 0.0
    out = ab.tp_forward(plan, rp, V, E, pw)
    gV, gE, _ = ab.tp_backward(plan, rp, out, V, E, pw)
    assert float(gE[0].abs().sum()) == 0.0 and float(gE[4].abs().sum()) == 0.0
    assert torch.isfinite(out).all() and torch.isfinite(gV).all() and torch.isfinite(gE).all()
    import oracle as orc
    ref = orc.tp_forward(2, rp.cpu().numpy(), V.cpu().numpy(), E.cpu().numpy(), pw.cpu().numpy())
    assert np.max(np.abs(ref - out.cpu().numpy())) <= 1e-5 * np.max(np.abs(ref))


def test_unsupported_and_bad_arguments_fail_loudly():
    import torch

    import paper_2504_16068_b200 as ab
    plan = ab.Plan(2, 3, ab.F32)      # 3 channels x 18 comps x 4 B = 216 B rows: not a multiple of 16
    rp = torch.tensor([0, 1], dtype=torch.int32, device="cuda")
    V = torch.zeros((1, 3, 18), device="cuda")
    E = torch.zeros((1, 3, 9), device="cuda")
    pw = torch.ones(30, device="cuda")
    with pytest.raises(ab.AllegroError) as ei:
        ab.tp_forward(plan, rp, V, E, pw)
    assert ei.value.status == 2
    plan = ab.Plan(2, 32, ab.F32)
    V = torch.zeros((1, 32, 18), device="cuda")
    E = torch.zeros((1, 32, 9), device="cuda")
    with pytest.raises(ab.AllegroError) as ei:
        ab.tp_forward(plan, rp, V, E, pw, out=V)      # aliasing
    assert ei.value.status == 1
    with pytest.raises(ab.AllegroError) as ei:        # workspace too small
        ab.tp_backward(plan, rp, V, V.clone(), E, pw, want_g_path_w=True, workspace=torch.empty(16, dtype=torch.uint8, device="cuda"))
    assert ei.value.status == 4
    # dense mix at l_max = 3: one n x n weight image must fit shared memory next to the staged tile (n <= 192 in fp32)
    dense = ab.Plan(3, 224, ab.F32, ab.W_DENSE)
    V3 = torch.zeros((1, 224, 32), device="cuda")
    E3 = torch.zeros((1, 224, 16), device="cuda")
    W3 = torch.zeros((68, 224, 224), device="cuda")
    with pytest.raises(ab.AllegroError) as ei:
        ab.tp_forward(dense, rp, V3, E3, W3)
    assert ei.value.status == 2 and "shared memory" in str(ei.value)
    with pytest.raises(ab.AllegroError) as ei:
        ab.tp_backward(dense, rp, V3, V3.clone(), E3, W3)
    assert ei.value.status == 2
    dense.set_out_blocks(0x1)                         # block subsets exist for the tensor-core shape only
    with pytest.raises(ab.AllegroError) as ei:
        ab.tp_forward(dense, rp, V3, E3, W3)
    assert ei.value.status == 2


def _check_sampled_centres(inp, got, ranges, label):
    """oracle on self-contained sub-problems (workloads.inputs.sub_inputs) vs the matching rows of the GPU result"""
    from workloads.inputs import sub_inputs
    edge_keys = ("w", "out", "e_edge", "G", "gV", "g_w", "g_r_env", "g_r")
    for c0, c1 in ranges:
        sub = sub_inputs(inp, c0, c1)
        ref = _chain.oracle_chain(sub, want_gw=False, forces=False)
        e0, e1 = sub["edge_range"]
        part = {k: got[k][e0:e1] for k in edge_keys if got.get(k) is not None}
        part.update(Eenv=got["Eenv"][c0:c1], gEenv=got["gEenv"][c0:c1])
        _assert_close(ref, part, inp["dt"], keys=edge_keys + ("Eenv", "gEenv"), label="%s centres [%d,%d)" % (label, c0, c1))


def _pool(fn, args_list, workers=None):
    """run fn over args_list on the host cores (the C++ oracle and torch release the GIL)"""
    import concurrent.futures as cf
    import os
    workers = workers or max(1, min(len(args_list), len(os.sched_getaffinity(0))))
    with cf.ThreadPoolExecutor(max_workers=workers) as ex:
        return list(ex.map(fn, args_list))


def _check_sampled_centres_pool(inp, got, ranges, label):
    """_check_sampled_centres with the oracle sub-problems fanned out over the host cores"""
    from workloads.inputs import sub_inputs
    edge_keys = ("w", "out", "e_edge", "G", "gV", "g_w", "g_r_env", "g_r")
    subs = [sub_inputs(inp, c0, c1) for c0, c1 in ranges]
    refs = _pool(lambda sb: _chain.oracle_chain(sb, want_gw=False, forces=False), subs)
    for (c0, c1), sub, ref in zip(ranges, subs, refs):
        e0, e1 = sub["edge_range"]
        part = {k: got[k][e0:e1] for k in edge_keys if got.get(k) is not None}
        part.update(Eenv=got["Eenv"][c0:c1], gEenv=got["gEenv"][c0:c1])
        _assert_close(ref, part, inp["dt"], keys=edge_keys + ("Eenv", "gEenv"), label="%s centres [%d,%d)" % (label, c0, c1))
    return sum(c1 - c0 for c0, c1 in ranges)


def _check_forces_vs_oracle(inp, F_gpu, atoms, g_r_of_centre, label):
    """Forces of `atoms` against the ORACLE's force assembly: atom a needs g_r of its own edges and of their reverses, i.e. the
    oracle's g_r rows of centre a and of every neighbour centre (each evaluated with its complete neighbourhood);
    F_ref[a] = sum_{e in row a} (g_r[e] - g_r[rev[e]]) in float64."""
    rp, rev = inp["row_ptr"], inp["rev"]
    centre_of = np.repeat(np.arange(inp["N"]), np.diff(rp))
    need = sorted({int(a) for a in atoms} | {int(centre_of[rev[e]]) for a in atoms for e in range(rp[a], rp[a + 1])})
    rows = dict(zip(need, _pool(g_r_of_centre, need)))
    Fref = np.zeros((len(atoms), 3))
    for i, a in enumerate(atoms):
        for e in range(rp[a], rp[a + 1]):
            j = int(centre_of[rev[e]])
            Fref[i] += rows[a][e - rp[a]] - rows[j][rev[e] - rp[j]]
    F = F_gpu[np.asarray(atoms)].detach().cpu().numpy().astype(np.float64)
    rel = np.linalg.norm(F - Fref) / np.linalg.norm(Fref)
    assert rel <= _chain.FORCE_RMS_TOL[inp["dt"]], "%s: forces of %d atoms vs oracle: relative RMS %g" % (label, len(atoms), rel)
    return rel


def _single_layer_g_r(inp):
    from workloads.inputs import sub_inputs
    return lambda c: _chain.oracle_chain(sub_inputs(inp, c, c + 1), want_gw=False, forces=False)["g_r"]


def _check_force_gather(inp, got):
    """F against a float64 host re-summation of the GPU's own g_r (integer gather + sum: size-independent property)"""
    g_r = got["g_r"].cpu().numpy().astype(np.float64)
    contrib = g_r - g_r[inp["rev"]]
    centre = np.repeat(np.arange(inp["N"]), np.diff(inp["row_ptr"]))
    Fref = np.zeros((inp["N"], 3))
    np.add.at(Fref, centre, contrib)
    F = got["F"].cpu().numpy().astype(np.float64)
    assert np.max(np.abs(F - Fref)) <= _chain.TOL[inp["dt"]] * np.max(np.abs(Fref))
    assert np.abs(F.sum(0)).max() <= 1e-3 * np.abs(F).max()


def test_c1_full_size_sampled_centres():
    """BASELINE.json:configs[1] at full size in the launch configuration bench.py times (V drawn in device memory);
    the oracle evaluates seeded centre ranges with their complete neighbourhoods, which is exact because every
    per-edge / per-centre output depends on one centre only."""
    from workloads import rng
    inp = _chain.make_inputs("C1", features="device")
    got = _chain.gpu_chain(inp, want_gw=False)
    N = inp["N"]
    starts = [int(x) for x in rng.randint(0, rng.STREAMS["sample"], np.arange(3), 0, N - 17)]
    deg = np.diff(inp["row_ptr"])
    ranges = [(c, c + 16) for c in starts + [0, N - 16]] + [(int(np.argmax(deg)), int(np.argmax(deg)) + 1), (int(np.argmin(deg)), int(np.argmin(deg)) + 1)]
    _check_sampled_centres_pool(inp, got, ranges, "C1")          # 2 % of the centres, the highest- and lowest-degree ones included
    _check_force_gather(inp, got)
    _check_forces_vs_oracle(inp, got["F"], [0, int(np.argmax(deg)), N - 1], _single_layer_g_r(inp), "C1")
    # the object bench.py times (preallocated buffers, fused forward + energy epilogue), same checks
    import paper_2504_16068_b200 as ab
    from paper_2504_16068_b200.pipeline import SingleLayerStep
    del got
    dev = _chain.to_device(inp)
    st = SingleLayerStep(ab.Plan(inp["lmax"], inp["n"], ab.F32), dev, inp["rc"], inp["kappa"], inp["scale"])
    st.run()
    got = dict(w=st.w, Eenv=st.Eenv, out=st.out, e_edge=st.e_edge, G=st.G, gV=st.gV, gEenv=st.gEenv, g_w=st.g_w, g_r=st.g_r, F=st.F)
    _check_sampled_centres(inp, got, ranges, "C1/SingleLayerStep")
    _check_force_gather(inp, got)
    e_tot = float(st.e_tot.item())
    e_ref = float(st.e_edge.double().sum().item())
    assert abs(e_tot - e_ref) <= 1e-5 * abs(e_ref)


def test_c4_full_size():
    """BASELINE.json:configs[4] in full (64 molecules, ~3k atoms, ~138k edges, l_max = 2, n = 32, fp32): forward, force VJP,
    path-weight gradient and per-molecule energies against the oracle, element by element"""
    inp = _chain.make_inputs("C4")
    ref = _chain.oracle_chain(inp)
    got = _chain.gpu_chain(inp)
    errs = _assert_close(ref, got, inp["dt"], label="C4")
    assert "E_mol" in errs and "g_path_w" in errs
    print("C4", {k: "%.2e" % v for k, v in errs.items()})


def test_c3_full_size_chunked_sampled_centres():
    """BASELINE.json:configs[3] at full size (100,000 atoms, ~5.2 M edges, l_max = 3, n = 128: 86 GB per feature tensor)
    through pipeline.ChunkedStep, the launch configuration bench.py --workload C3 times; the oracle evaluates seeded
    centre ranges with their complete neighbourhoods (exact: strict locality) inside the first, a middle and the last chunk"""
    import torch

    import paper_2504_16068_b200 as ab
    from paper_2504_16068_b200.pipeline import ChunkedStep, to_device
    from workloads.inputs import sub_inputs
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 140e9:
        pytest.skip("needs ~135 GB of free HBM")
    inp = _chain.make_inputs("C3", features="device")
    dev = to_device(inp)
    plan = ab.Plan(inp["lmax"], inp["n"], ab.F32)
    st = ChunkedStep(plan, dev, inp["row_ptr"], inp["rc"], inp["kappa"], inp["scale"], n_chunks=16)
    nck = len(st.chunks)
    # ~2 % of the centres: in EVERY chunk a window at its first centres, at its middle and at its last centres (both
    # sides of every chunk boundary), plus the highest- and the lowest-degree centre of the system
    W = 40
    rp = inp["row_ptr"]
    deg = np.diff(rp)
    windows = {k: [] for k in range(nck)}
    for k, (c0, c1, e0, e1, _) in enumerate(st.chunks):
        for a in (c0, (c0 + c1) // 2, c1 - W):
            windows[k].append((a, a + W))
    for c in (int(np.argmax(deg)), int(np.argmin(deg))):
        k = next(i for i, ch in enumerate(st.chunks) if ch[0] <= c < ch[1])
        windows[k].append((c, c + 1))
    keep = {k: {"rows": [(int(rp[a]), int(rp[b])) for a, b in ws]} for k, ws in windows.items()}
    st.run(keep=keep)
    torch.cuda.synchronize()
    jobs = [(k, i, a, b) for k, ws in windows.items() for i, (a, b) in enumerate(ws)]
    subs = [sub_inputs(inp, a, b) for _, _, a, b in jobs]
    refs = _pool(lambda sb: _chain.oracle_chain(sb, want_gw=False, forces=False), subs)
    n_checked = 0
    for (k, i, a, b), sub, ref in zip(jobs, subs, refs):
        s0, s1 = sub["edge_range"]
        part = dict(out=keep[k]["out"][i], gV=keep[k]["gV"][i], e_edge=st.e_edge[s0:s1], g_r=st.g_r[s0:s1], Eenv=st.Eenv[a:b], gEenv=st.gEenv[a:b])
        _assert_close(ref, part, inp["dt"], keys=tuple(part.keys()), label="C3 chunk %d centres [%d,%d)" % (k, a, b))
        n_checked += b - a
    assert n_checked >= 0.019 * inp["N"]
    got = dict(g_r=st.g_r, F=st.F)
    _check_force_gather(inp, got)
    _check_forces_vs_oracle(inp, st.F, [0, int(np.argmax(deg)), inp["N"] - 1], _single_layer_g_r(inp), "C3")


@pytest.mark.parametrize("lmax,n,dt,geom", [(2, 64, np.float32, "C1s"), (1, 8, np.float64, "C0"), (1, 128, np.float32, "C0"), (2, 32, np.float64, "C4s"),
                                            (3, 128, np.float32, "C0"), (3, 64, np.float32, "C0"), (3, 16, np.float64, "C0")])
def test_dense_path_weights_forward_and_vjp(lmax, n, dt, geom):
    """ALLEGRO_W_DENSE (BASELINE.json:configs[2], reading A5): per-path n x n channel mix, forward and VJP (gV, gEenv),
    against the oracle's dense mode on seeded inputs; also with centres split into items.  l_max = 3 (Table 1's medium / large
    models: 68 paths, n = 64 / 128) runs the paths-outer kernels."""
    import oracle as orc
    import torch

    import paper_2504_16068_b200 as ab
    from workloads import configs, rng
    g = configs.geometry_for(geom)
    rp, E, N = g["row_ptr"], g["rvec"].shape[0], g["row_ptr"].shape[0] - 1
    dV, dE, P = 2 * (lmax + 1) ** 2, (lmax + 1) ** 2, configs.num_paths(lmax)
    S = rng.STREAMS
    V = rng.normal(7, S["V"], (E, n, dV)).astype(dt)
    Ee = (rng.normal(7, S["W_w"], (N, n, dE)) * 0.5).astype(dt)
    W = (rng.normal(7, S["W_p"], (P, n, n)) / np.sqrt(n)).astype(dt)
    G = rng.normal(7, S["G"], (E, n, dV)).astype(dt)
    f8 = lambda a: a.astype(np.float64)
    ref_out = orc.tp_forward(lmax, rp, f8(V), f8(Ee), f8(W))
    ref_gV, ref_gE, ref_gW = orc.tp_backward(lmax, rp, f8(G), f8(V), f8(Ee), f8(W), want_gV=True, want_gw=True)
    assert ref_gW.shape == W.shape
    plan = ab.Plan(lmax, n, ab.F64 if dt == np.float64 else ab.F32, ab.W_DENSE)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    rpd, Vd, Ed, Wd, Gd = d(rp), d(V), d(Ee), d(W), d(G)
    for items in (None, ab.segments_build(rp, 6)):
        it = None if items is None else d(items)
        out = ab.tp_forward(plan, rpd, Vd, Ed, Wd, items=it)
        gV, gE, gW = ab.tp_backward(plan, rpd, Gd, Vd, Ed, Wd, items=it, want_g_path_w=True)      # training: dE/dW_p as well (row f2)
        _assert_close(dict(out=ref_out, gV=ref_gV, gEenv=ref_gE, g_path_w=ref_gW), dict(out=out, gV=gV, gEenv=gE, g_path_w=gW), dt,
                      keys=("out", "gV", "gEenv", "g_path_w"), label="dense l%d n%d" % (lmax, n))
        gW2 = ab.tp_backward(plan, rpd, Gd, Vd, Ed, Wd, items=it, want_g_path_w=True)[2]
        assert torch.equal(gW, gW2)                                                             # fixed-order reduction: reproducible bits
        _, gE2, _ = ab.tp_backward(plan, rpd, Gd, Vd, Ed, Wd, items=it, want_gV=False)
        _assert_close(dict(gEenv=ref_gE), dict(gEenv=gE2), dt, keys=("gEenv",), label="dense force-only")
        if lmax == 2 and n == 64 and dt == np.float32:
            # compact side channel of the 0e scalars (allegro_tp_forward_aux / _backward_aux): bitwise the plain calls' results
            out2, sc = torch.empty_like(out), torch.empty((E, n, 1), dtype=out.dtype, device="cuda")
            ab.tp_forward_aux(plan, rpd, Vd, Ed, Wd, out2, sc, items=it)
            assert torch.equal(out2, out) and torch.equal(sc[:, :, 0], out[:, :, 0])
            gs = torch.from_numpy(rng.normal(8, S["q"], (E, n, 1)).astype(dt)).cuda()
            G2 = Gd.clone()
            G2[:, :, 0] += gs[:, :, 0]
            gV_a, gE_a, _ = ab.tp_backward(plan, rpd, G2, Vd, Ed, Wd, items=it)
            gV_b, gE_b = ab.tp_backward_aux(plan, rpd, Gd, gs, Vd, Ed, Wd, torch.empty_like(Vd), torch.empty_like(Ed), items=it)
            assert torch.equal(gV_a, gV_b) and torch.equal(gE_a, gE_b)


def _block_mask_weights(lmax, W, out_mask, in_mask=0xffff):
    """path weights with the paths into blocks outside out_mask / from blocks outside in_mask zeroed: what a block subset computes"""
    import oracle as orc
    pt = orc.paths(lmax)
    Wm = np.array(W, copy=True)
    for p in range(len(pt["l3"])):
        if not ((out_mask >> (2 * int(pt["l3"][p]) + int(pt["p3"][p]))) & 1 and (in_mask >> (2 * int(pt["l1"][p]) + int(pt["p1"][p]))) & 1):
            Wm[p] = 0
    return Wm


@pytest.mark.parametrize("wmode", ["dense", "scalar"])
def test_input_block_subset(wmode):
    """allegro_plan_set_in_blocks(0x19): V has the natural-parity blocks (0e, 1o, 2e) only -- the first layer of the two-layer
    model, V0 = v (x) Y.  The other blocks of V are never read (they hold garbage here), the paths from them never run, their gV
    components come back as zeros; everything else equals the oracle on V with those blocks zeroed."""
    import oracle as orc
    import torch

    import paper_2504_16068_b200 as ab
    from workloads import configs, rng
    lmax, n, dt = 2, 64, np.float32
    g = configs.geometry_for("C1s")
    rp, E, N = g["row_ptr"], g["rvec"].shape[0], g["row_ptr"].shape[0] - 1
    dV, dE, P = 18, 9, 30
    S = rng.STREAMS
    V = rng.normal(13, S["V"], (E, n, dV)).astype(dt)
    Ee = (rng.normal(13, S["W_w"], (N, n, dE)) * 0.5).astype(dt)
    W = (rng.normal(13, S["W_p"], (P, n, n)) / np.sqrt(n)).astype(dt) if wmode == "dense" else rng.normal(13, S["path_w"], (P,)).astype(dt)
    G = rng.normal(13, S["G"], (E, n, dV)).astype(dt)
    natural = [0, 5, 6, 7, 8, 9, 10, 11, 12]                  # components of 0e, 1o, 2e
    other = [k for k in range(dV) if k not in natural]
    Vz = V.copy()
    Vz[:, :, other] = 0
    f8 = lambda a: a.astype(np.float64)
    ref_out = orc.tp_forward(lmax, rp, f8(Vz), f8(Ee), f8(W))
    ref_gV, ref_gE, _ = orc.tp_backward(lmax, rp, f8(G), f8(Vz), f8(Ee), f8(W), want_gV=True, want_gw=False)
    ref_gV[:, :, other] = 0
    plan = ab.Plan(lmax, n, ab.F32, ab.W_DENSE if wmode == "dense" else ab.W_SCALAR)
    plan.set_in_blocks(0x19)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    Vg = V.copy()
    Vg[:, :, other] = 1e30                                    # must never be read
    rpd, Vd, Ed, Wd, Gd = d(rp), d(Vg), d(Ee), d(W), d(G)
    for items in (None, ab.segments_build(rp, 30)):
        it = None if items is None else d(items)
        out = ab.tp_forward(plan, rpd, Vd, Ed, Wd, items=it)
        gV, gE, _ = ab.tp_backward(plan, rpd, Gd, Vd, Ed, Wd, items=it)
        _assert_close(dict(out=ref_out, gV=ref_gV, gEenv=ref_gE), dict(out=out, gV=gV, gEenv=gE), dt, keys=("out", "gV", "gEenv"),
                      label="natural-parity inputs " + wmode)
        assert float(gV[:, :, other].abs().max().item()) == 0.0


@pytest.mark.parametrize("wmode", ["dense", "scalar"])
def test_output_block_subset(wmode):
    """allegro_plan_set_out_blocks(0x1): only the paths into the 0e scalars run (last layer of a model whose readout takes the
    l = 0 outputs, BASELINE.json:configs[2]).  Forward and VJP equal the oracle evaluated with the other paths' weights set
    to zero; the cotangent outside the block is ignored."""
    import oracle as orc
    import torch

    import paper_2504_16068_b200 as ab
    from workloads import configs, rng
    lmax, n, dt = 2, 64, np.float32
    g = configs.geometry_for("C1s")
    rp, E, N = g["row_ptr"], g["rvec"].shape[0], g["row_ptr"].shape[0] - 1
    dV, dE, P = 18, 9, 30
    S = rng.STREAMS
    V = rng.normal(11, S["V"], (E, n, dV)).astype(dt)
    Ee = (rng.normal(11, S["W_w"], (N, n, dE)) * 0.5).astype(dt)
    W = (rng.normal(11, S["W_p"], (P, n, n)) / np.sqrt(n)).astype(dt) if wmode == "dense" else rng.normal(11, S["path_w"], (P,)).astype(dt)
    G = rng.normal(11, S["G"], (E, n, dV)).astype(dt)
    f8 = lambda a: a.astype(np.float64)
    Wm = _block_mask_weights(lmax, W, 0x1)
    Gm = np.zeros_like(G)
    Gm[:, :, 0] = G[:, :, 0]
    ref_out = orc.tp_forward(lmax, rp, f8(V), f8(Ee), f8(Wm))
    ref_gV, ref_gE, _ = orc.tp_backward(lmax, rp, f8(Gm), f8(V), f8(Ee), f8(Wm), want_gV=True, want_gw=False)
    assert np.abs(ref_out[:, :, 1:]).max() == 0.0
    plan = ab.Plan(lmax, n, ab.F32, ab.W_DENSE if wmode == "dense" else ab.W_SCALAR)
    plan.set_out_blocks(0x1)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    rpd, Vd, Ed, Wd, Gd = d(rp), d(V), d(Ee), d(W), d(G)
    for items in (None, ab.segments_build(rp, 30)):
        it = None if items is None else d(items)
        out = ab.tp_forward(plan, rpd, Vd, Ed, Wd, items=it)
        gV, gE, _ = ab.tp_backward(plan, rpd, Gd, Vd, Ed, Wd, items=it)     # full G handed in: its other blocks must be ignored
        _assert_close(dict(out=ref_out, gV=ref_gV, gEenv=ref_gE), dict(out=out, gV=gV, gEenv=gE), dt, keys=("out", "gV", "gEenv"),
                      label="0e-only " + wmode)
        assert float(out[:, :, 1:].abs().max().item()) == 0.0
    if wmode == "dense":
        # energy epilogue of the dense forward (e_edge formed from the rows in registers; `out` optional) and the VJP whose cotangent
        # q (x) delta + kappa out is formed while staging (no `out` read at all when kappa = 0)
        q = (rng.normal(11, S["q"], (n,)) / np.sqrt(n)).astype(dt)
        qd = d(q)
        for kappa in (0.3, 0.0):
            e_ref, G_ref = orc.edge_energy(lmax, ref_out, f8(q), kappa)
            Gm2 = np.zeros_like(G_ref)
            Gm2[:, :, 0] = G_ref[:, :, 0]
            gV_ref, gE_ref, _ = orc.tp_backward(lmax, rp, Gm2, f8(V), f8(Ee), f8(Wm), want_gV=True, want_gw=False)
            o2, e2, _ = ab.tp_forward_energy(plan, rpd, Vd, Ed, Wd, qd, kappa, want_out=(kappa != 0.0), want_G=False)
            gV2, gE2, _ = ab.tp_backward_energy(plan, rpd, o2, Vd, Ed, Wd, qd, kappa)
            _assert_close(dict(e_edge=e_ref, gV=gV_ref, gEenv=gE_ref), dict(e_edge=e2, gV=gV2, gEenv=gE2), dt, keys=("e_edge", "gV", "gEenv"),
                          label="dense energy epilogue kappa=%g" % kappa)
        plan.set_out_blocks(0x5)      # not a compiled subset
        with pytest.raises(ab.AllegroError) as ei:
            ab.tp_forward(plan, rpd, Vd, Ed, Wd)
        assert ei.value.status == 2


def test_two_plans_two_streams_concurrently():
    """Two plans of the same dtype / l_max with different scalar path weights, run on two streams at the same time: the folded
    coefficient table travels with each launch as a kernel parameter, so neither sees the other's weights (round-1 finding:
    a process-global __constant__ table raced).  Both results against the oracle."""
    import oracle as orc
    import torch

    import paper_2504_16068_b200 as ab
    from workloads import rng
    inp = _chain.make_inputs("C1s")
    lmax, n, rp = inp["lmax"], inp["n"], inp["row_ptr"]
    dev = _chain.to_device(inp)
    f8 = lambda a: np.asarray(a, dtype=np.float64)
    w, _ = orc.radial(f8(inp["W_r"]), inp["rc"], f8(inp["rvec"]))
    Eenv = orc.env_embed(lmax, rp, f8(inp["rvec"]), w, inp["scale"])
    Ed = torch.from_numpy(Eenv.astype(np.float32)).cuda()
    Eenv = f8(Ed.cpu().numpy())
    pws = [inp["path_w"], rng.normal(3, rng.STREAMS["path_w"], inp["path_w"].shape).astype(np.float32)]
    refs = [orc.tp_forward(lmax, rp, f8(inp["V"]), Eenv, f8(pw)) for pw in pws]
    plans = [ab.Plan(lmax, n, ab.F32), ab.Plan(lmax, n, ab.F32)]
    pwd = [torch.from_numpy(pw).cuda() for pw in pws]
    for pl, pw in zip(plans, pwd):
        pl.bind_weights(pw)
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    outs = [torch.empty_like(dev["V"]) for _ in range(2)]
    torch.cuda.synchronize()
    for rep in range(20):          # interleaved launches, no host synchronisation in between
        for k in range(2):
            with torch.cuda.stream(streams[k]):
                ab.tp_forward(plans[k], dev["row_ptr"], dev["V"], Ed, None, out=outs[k], stream=streams[k])
    torch.cuda.synchronize()
    for k in range(2):
        _assert_close(dict(out=refs[k]), dict(out=outs[k]), np.float32, keys=("out",), label="plan %d" % k)
    assert not torch.equal(outs[0], outs[1])
    # a call without bound weights and without path_w fails loudly
    with pytest.raises(ab.AllegroError) as ei:
        ab.tp_forward(ab.Plan(lmax, n, ab.F32), dev["row_ptr"], dev["V"], Ed, None)
    assert ei.value.status == 1


@pytest.mark.parametrize("n,dt", [(48, np.float32), (96, np.float32), (48, np.float64), (96, np.float64), (160, np.float32)])
def test_energy_epilogue_channel_counts(n, dt):
    """tp_forward_energy / tp_backward_energy for channel counts that leave compute threads without an edge slot (256 % 96 != 0)
    or take the serial per-edge sum (n = 48): e_edge, out, gV, gEenv against the oracle (round-1 finding: n = 96 hung)."""
    import oracle as orc
    import torch

    import paper_2504_16068_b200 as ab
    from workloads import configs, rng
    lmax = 1
    g = configs.geometry_for("C0")
    rp, E, N = g["row_ptr"], g["rvec"].shape[0], g["row_ptr"].shape[0] - 1
    dV, dE, P = 8, 4, 10
    S = rng.STREAMS
    V = rng.normal(5, S["V"], (E, n, dV)).astype(dt)
    Ee = (rng.normal(5, S["W_w"], (N, n, dE)) * 0.5).astype(dt)
    pw = rng.normal(5, S["path_w"], (P,)).astype(dt)
    q = (rng.normal(5, S["q"], (n,)) / np.sqrt(n)).astype(dt)
    kappa = 0.3
    f8 = lambda a: a.astype(np.float64)
    out = orc.tp_forward(lmax, rp, f8(V), f8(Ee), f8(pw))
    e_edge, G = orc.edge_energy(lmax, out, f8(q), kappa)
    gV, gE, _ = orc.tp_backward(lmax, rp, G, f8(V), f8(Ee), f8(pw), want_gV=True, want_gw=False)
    plan = ab.Plan(lmax, n, ab.F64 if dt == np.float64 else ab.F32)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    rpd, Vd, Ed, pwd, qd = d(rp), d(V), d(Ee), d(pw), d(q)
    o, e, Gd = ab.tp_forward_energy(plan, rpd, Vd, Ed, pwd, qd, kappa)
    gVd, gEd, _ = ab.tp_backward_energy(plan, rpd, o, Vd, Ed, pwd, qd, kappa)
    torch.cuda.synchronize()
    _assert_close(dict(out=out, e_edge=e_edge, G=G, gV=gV, gEenv=gE), dict(out=o, e_edge=e, G=Gd, gV=gVd, gEenv=gEd), dt,
                  keys=("out", "e_edge", "G", "gV", "gEenv"), label="n=%d" % n)
    # the same through the single fused kernel (forward + energy + VJP), also with centres split into items
    for items in (None, ab.segments_build(rp, 5)):
        it = None if items is None else d(items)
        e2, gV2, gE2, _ = ab.tp_fused_energy(plan, rpd, Vd, Ed, pwd, qd, kappa, items=it)
        torch.cuda.synchronize()
        _assert_close(dict(e_edge=e_edge, gV=gV, gEenv=gE), dict(e_edge=e2, gV=gV2, gEenv=gE2), dt, keys=("e_edge", "gV", "gEenv"), label="fused n=%d" % n)


def _model_device(inp):
    import torch
    td = torch.float32 if inp["dt"] == np.float32 else torch.float64
    p = inp["params"]
    dev = {k: torch.from_numpy(np.ascontiguousarray(inp[k])).cuda() for k in ("row_ptr", "rev", "rvec")}
    prm = {k: torch.from_numpy(np.ascontiguousarray(p[k])).to(td).cuda() for k in ("W_x0", "W_v0", "W_w", "W_p", "A_lat", "q")}
    prm.update(rc=p["rc"], scale=p["scale"])
    return dev, prm


def _two_layer_step(inp, scalars_only_last=False):
    import paper_2504_16068_b200 as ab
    from paper_2504_16068_b200.pipeline import TwoLayerStep
    p = inp["params"]
    dt = ab.F32 if inp["dt"] == np.float32 else ab.F64
    dev, prm = _model_device(inp)
    last = first = None
    if scalars_only_last:      # the launch configuration bench.py --workload C2 times: block subsets for the first and last layer
        last = ab.Plan(p["lmax"], p["n"], dt, ab.W_DENSE)
        last.set_out_blocks(0x1)
        first = ab.Plan(p["lmax"], p["n"], dt, ab.W_DENSE)
        first.set_in_blocks(0x19)
    st = TwoLayerStep(ab.Plan(p["lmax"], p["n"], dt, ab.W_DENSE), ab.Plan(p["lmax"], p["n"], dt, ab.W_SCALAR), dev, prm, plan_last=last,
                      plan_first=first, fuse_readout=(scalars_only_last == "fused_readout"), factorised_env=bool(scalars_only_last))
    st.run()
    return st


@pytest.mark.parametrize("scalars_only_last", [False, True, "fused_readout"])
def test_two_layer_model_c2s(scalars_only_last):
    """BASELINE.json:configs[2]'s recipe at 192 atoms (two stacked layers, dense 64x64 per-path mix, latent update, readout of
    the l = 0 outputs; forward + force backward) against oracle/model2.py: per-layer Eenv and features, per-edge energies,
    total energy, dE/dr_e and forces"""
    from oracle import model2
    import oracle as orc
    from workloads.inputs import make_model_inputs
    inp = make_model_inputs("C2s")
    p = inp["params"]
    taps = []
    en, g = model2.energy_grad(p, inp["row_ptr"], inp["rvec"].astype(np.float64), taps)
    st = _two_layer_step(inp, scalars_only_last)
    ref, got = dict(g_r=g, e_edge=taps[-1]["e_edge"], F=orc.force_gather(inp["row_ptr"], inp["rev"], g)), dict(g_r=st.g_r, e_edge=st.e_edge, F=st.F)
    for l in range(p["n_layers"]):
        ref.update({"Eenv%d" % l: taps[l]["Eenv"], "V%d" % (l + 1): taps[l]["V_out"]})
        got.update({"Eenv%d" % l: st.Eenv[l], "V%d" % (l + 1): st.V[l + 1]})
        if not st.factorised_env:      # the per-edge weights w = W_w x exist only on the un-factorised path
            ref["w%d" % l], got["w%d" % l] = taps[l]["w"], st.w[l]
    if scalars_only_last:      # only the scalars of the last layer's output exist
        L = p["n_layers"]
        if st.V[L] is None:    # readout fused into the last layer's forward: V_L is never stored
            ref.pop("V%d" % L), got.pop("V%d" % L)
        else:
            ref["V%d" % L], got["V%d" % L] = taps[L - 1]["V_out"][:, :, :1], st.V[L][:, :, :1]
    ref["V0"], got["V0"] = taps[0]["V_in"], st.V[0]
    errs = _assert_close(ref, got, inp["dt"], keys=tuple(ref.keys()), label="C2s")
    print("C2s", {k: "%.2e" % v for k, v in errs.items()})
    assert abs(float(st.e_tot.item()) - en) <= 1e-5 * max(abs(en), float(np.abs(taps[-1]["e_edge"]).max()))
    F = st.F.cpu().numpy().astype(np.float64)
    assert np.abs(F.sum(0)).max() <= 1e-3 * np.abs(F).max()


def test_two_layer_model_c2_full_size_sampled_centres():
    """configs[2] at full size (32,768 atoms, ~2.95 M edges) in the launch configuration bench.py --workload C2 times;
    the oracle evaluates seeded centre ranges with their complete neighbourhoods (exact: the model is strictly local)"""
    import torch
    from oracle import model2
    from workloads import rng
    from workloads.inputs import make_model_inputs
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 110e9:
        pytest.skip("needs ~100 GB of free HBM")
    inp = make_model_inputs("C2")
    st = _two_layer_step(inp, scalars_only_last="fused_readout")      # the launch configuration bench.py --workload C2 times
    torch.cuda.synchronize()
    rp, N = inp["row_ptr"], inp["N"]
    deg = np.diff(rp)
    # ~1 % of the centres: 80 seeded windows of 4 centres, both ends of the system, the highest- and lowest-degree centre
    starts = sorted({int(x) for x in rng.randint(0, rng.STREAMS["sample"], np.arange(80), 0, N - 5)} | {0, N - 4})
    ranges = [(c, c + 4) for c in starts] + [(int(np.argmax(deg)), int(np.argmax(deg)) + 1), (int(np.argmin(deg)), int(np.argmin(deg)) + 1)]

    def oracle_range(cr):
        c0, c1 = cr
        e0, e1 = int(rp[c0]), int(rp[c1])
        taps = []
        en, g = model2.energy_grad(inp["params"], (rp[c0:c1 + 1] - rp[c0]).astype(np.int32), inp["rvec"][e0:e1].astype(np.float64), taps)
        return g, taps

    refs = _pool(oracle_range, ranges, workers=4)      # model2 is multi-threaded torch: a few ranges at a time
    n_checked = 0
    for (c0, c1), (g, taps) in zip(ranges, refs):
        e0, e1 = int(rp[c0]), int(rp[c1])
        ref = dict(g_r=g, e_edge=taps[-1]["e_edge"], V1=taps[0]["V_out"], Eenv1=taps[1]["Eenv"])
        got = dict(g_r=st.g_r[e0:e1], e_edge=st.e_edge[e0:e1], V1=st.V[1][e0:e1], Eenv1=st.Eenv[1][c0:c1])
        _assert_close(ref, got, inp["dt"], keys=tuple(ref.keys()), label="C2 centres [%d,%d)" % (c0, c1))
        n_checked += c1 - c0
    assert n_checked >= 0.0095 * N
    _check_force_gather(inp, dict(g_r=st.g_r, F=st.F))
    _check_forces_vs_oracle(inp, st.F, [0, N - 1], lambda c: oracle_range((c, c + 1))[0], "C2")


@pytest.mark.parametrize("name", ["C0", "C1s"])
def test_host_buffer_step_through_c_abi(name):
    """allegro_layer_step_host: host buffers in, forces and total energy out in one C-ABI call (bench.py's end-to-end arm)"""
    import torch

    import paper_2504_16068_b200 as ab
    from paper_2504_16068_b200.pipeline import HostStep, SingleLayerStep
    inp = _chain.make_inputs(name)
    ref = _chain.oracle_chain(inp, want_gw=False)
    plan = ab.Plan(inp["lmax"], inp["n"], ab.F64 if inp["dt"] == np.float64 else ab.F32)
    st = SingleLayerStep(plan, _chain.to_device(inp), inp["rc"], inp["kappa"], inp["scale"])
    hs = HostStep(st)
    F, e = hs.run()
    _assert_close(ref, dict(F=F), inp["dt"], keys=("F",), label=name + "/host")
    e_ref = float(np.sum(ref["e_edge"]))
    assert abs(float(e.item()) - e_ref) <= _chain.TOL[inp["dt"]] * max(abs(e_ref), float(np.abs(ref["e_edge"]).max()))
    with pytest.raises(ab.AllegroError) as ei:
        ab.layer_step_host(plan, hs.host["row_ptr"], hs.host["rev"], hs.host["rvec"], hs.host["V"], hs.host["W_r"], inp["rc"], hs.host["path_w"],
                           hs.host["q"], inp["kappa"], inp["scale"], hs.F_host, hs.e_host, torch.empty(256, dtype=torch.uint8, device="cuda"))
    assert ei.value.status == 4


def test_cuda_graph_replay_matches_eager():
    """pipeline.GraphedStep: the step captured into one CUDA graph gives the same bits as the eager call sequence, also after
    the inputs change in place (an MD loop updates rvec between steps)"""
    import torch

    import paper_2504_16068_b200 as ab
    from paper_2504_16068_b200.pipeline import GraphedStep, SingleLayerStep
    inp = _chain.make_inputs("C4s")
    dev = _chain.to_device(inp)
    plan = ab.Plan(inp["lmax"], inp["n"], ab.F32)
    st = SingleLayerStep(plan, dev, inp["rc"], inp["kappa"], inp["scale"])
    st.run()
    F0, e0 = st.F.clone(), st.e_tot.clone()
    gs = GraphedStep(st)
    st.F.zero_()
    gs.run()
    torch.cuda.synchronize()
    assert torch.equal(gs.F, F0) and torch.equal(gs.e_tot, e0)
    dev["rvec"].mul_(1.01)                       # new geometry, same graph
    gs.run()
    F1 = gs.F.clone()
    st.run()
    torch.cuda.synchronize()
    assert torch.equal(st.F, F1) and not torch.equal(F1, F0)


def test_sharded_step_single_rank_matches_unsharded():
    """pipeline / sharding binding on the GPU with a one-rank process group (the box has one GPU): ShardedForces' index arrays,
    the extended g_r array and the owner's force gather give bitwise the forces of the unsharded step; the multi-rank exchange
    itself is covered on CPU by tests/test_sharding_gloo.py (world_size 2 and 3, bitwise against the oracle)."""
    import os

    import torch
    import torch.distributed as dist

    import paper_2504_16068_b200 as ab
    from paper_2504_16068_b200.pipeline import SingleLayerStep, shard_to_device
    from paper_2504_16068_b200.sharding import ShardedForces
    inp = _chain.make_inputs("C1s")
    plan = ab.Plan(inp["lmax"], inp["n"], ab.F32)
    st0 = SingleLayerStep(plan, _chain.to_device(inp), inp["rc"], inp["kappa"], inp["scale"])
    st0.run()
    created = False
    if not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", str(29600 + os.getpid() % 2000))
        dist.init_process_group("gloo", rank=0, world_size=1)
        created = True
    try:
        sh = ShardedForces(inp["row_ptr"], inp["rev"], device="cuda", dtype=torch.float32)
        dev = shard_to_device(inp, sh)
        st1 = SingleLayerStep(plan, dev, inp["rc"], inp["kappa"], inp["scale"], sharded=sh)
        st1.run(mark=True)
        torch.cuda.synchronize()
        assert torch.equal(st1.F, st0.F) and torch.equal(st1.e_tot, st0.e_tot) and torch.equal(st1.g_r, st0.g_r)
        assert {"halo_exchange", "energy_all_reduce"} <= {nm for nm, _, _ in st1.marks}
    finally:
        if created:
            dist.destroy_process_group()


@pytest.mark.parametrize("name", ["C0", "C4s"])
def test_library_graph_step_matches_eager(name):
    """allegro_layer_step_create / _launch: the step captured into a CUDA graph INSIDE the library (no torch graph, one launch per
    MD step) gives the bits of the eager call sequence, also after the edge vectors change in place; buffers are reachable"""
    import torch

    import paper_2504_16068_b200 as ab
    from paper_2504_16068_b200.pipeline import SingleLayerStep
    inp = _chain.make_inputs(name)
    dev = _chain.to_device(inp)
    dt = ab.F64 if inp["dt"] == np.float64 else ab.F32
    plan = ab.Plan(inp["lmax"], inp["n"], dt)
    st = SingleLayerStep(plan, dev, inp["rc"], inp["kappa"], inp["scale"])
    st.run()
    F0, e0, gV0 = st.F.clone(), st.e_tot.clone(), st.gV.clone()
    F, e = torch.empty_like(st.F), torch.empty_like(st.e_tot)
    g = ab.LayerStepGraph(plan, dev["row_ptr"], dev["rev"], dev["rvec"], dev["V"], dev["W_r"], inp["rc"], dev["q"], inp["kappa"], inp["scale"], F, e)
    assert g.kernels_per_step == 5
    F.zero_()
    g.run()
    torch.cuda.synchronize()
    assert torch.equal(F, F0) and torch.equal(e, e0)
    assert torch.equal(g.buffer("gV", tuple(st.gV.shape), st.gV.dtype), gV0)
    dev["rvec"].mul_(1.01)
    g.run()
    st.run()
    torch.cuda.synchronize()
    assert torch.equal(F, st.F) and not torch.equal(F, F0)
    with pytest.raises(ab.AllegroError) as ei:          # weights must be bound before the capture
        ab.LayerStepGraph(ab.Plan(inp["lmax"], inp["n"], dt), dev["row_ptr"], dev["rev"], dev["rvec"], dev["V"], dev["W_r"], inp["rc"], dev["q"],
                          inp["kappa"], inp["scale"], F, e)
    assert ei.value.status == 1


@pytest.mark.parametrize("name", ["C0", "C1s", "C4s"])
def test_virial(name):
    """allegro_virial against the oracle's (reading A25), on the g_r of the GPU chain; bitwise reproducible"""
    import oracle as orc
    import torch

    import paper_2504_16068_b200 as ab
    inp = _chain.make_inputs(name)
    got = _chain.gpu_chain(inp, want_gw=False)
    dev = _chain.to_device(inp)
    W = ab.virial(dev["rvec"], got["g_r"])
    ref = orc.virial(inp["rvec"].astype(np.float64), got["g_r"].cpu().numpy().astype(np.float64))
    assert np.max(np.abs(W.cpu().numpy().astype(np.float64) - ref)) <= _chain.TOL[inp["dt"]] * np.max(np.abs(ref))
    assert torch.equal(W, ab.virial(dev["rvec"], got["g_r"]))
    ref_full = orc.virial(inp["rvec"].astype(np.float64), _chain.oracle_chain(inp, want_gw=False, forces=False)["g_r"])
    assert np.max(np.abs(W.cpu().numpy().astype(np.float64) - ref_full)) <= 10 * _chain.TOL[inp["dt"]] * np.max(np.abs(ref_full))


@pytest.mark.parametrize("name", ["C0", "C1s", "C4s", "C1"])
def test_gpu_neighbour_list_bit_exact(name):
    """allegro_neighbour_count / _fill: the cell-list builder on the GPU gives the CSR list of workloads/geometry.py (k-d tree on the
    host) bit for bit -- row_ptr, neighbour indices, reverse-edge permutation -- and the same edge vectors after the one rounding
    to the config's dtype (readings A7, A9, A17); C0's box holds two cells per direction (all-pairs path), C4s is open with a
    molecule filter, C1 is the full 4,096-atom box"""
    import torch

    import paper_2504_16068_b200 as ab
    from workloads import configs
    g = configs.geometry_for(name)
    dt = np.float64 if g["spec"]["dtype"] == "f64" else np.float32
    pos = torch.from_numpy(np.ascontiguousarray(g["pos"])).cuda()
    mol = None
    if g["mol_ptr"] is not None:
        mol = torch.from_numpy((np.searchsorted(g["mol_ptr"], np.arange(pos.shape[0]), side="right") - 1).astype(np.int32)).cuda()
    nl = ab.neighbour_list(pos, g["spec"]["rc"], box=g["box"], mol_id=mol, dtype=ab.F64 if dt == np.float64 else ab.F32)
    torch.cuda.synchronize()
    assert np.array_equal(nl["row_ptr"].cpu().numpy(), g["row_ptr"])
    assert np.array_equal(nl["col"].cpu().numpy(), g["col"])
    assert np.array_equal(nl["rev"].cpu().numpy(), g["rev"])
    assert np.array_equal(nl["rvec"].cpu().numpy(), g["rvec"].astype(dt))


@pytest.mark.parametrize("n_in,n_out", [(64, 64), (64, 128), (32, 64)])
def test_linear_map_and_its_transpose(n_in, n_out):
    """allegro_linear: y (+)= x W^T and the transposed map with accumulation (the per-edge linear of reading A19 and its VJP), against the
    float64 matrix products.  fp32 with 64 inputs and 64 outputs runs on tcgen05 (tclin.cu), the other shapes on the FMA tiles;
    333 rows = two full 128-row tiles and a ragged one"""
    import torch

    import paper_2504_16068_b200 as ab
    from workloads import rng
    S = rng.STREAMS
    R = 333
    x = rng.normal(61, S["V"], (R, n_in)).astype(np.float32)
    W = (rng.normal(62, S["W_p"], (n_out, n_in)) / np.sqrt(n_in)).astype(np.float32)
    g = rng.normal(63, S["G"], (R, n_out)).astype(np.float32)
    y0 = rng.normal(64, S["q"], (R, n_in)).astype(np.float32)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    f8 = lambda a: a.astype(np.float64)
    y = ab.linear(d(x), d(W))
    gx = ab.linear(d(g), d(W), transpose_w=True)
    acc = d(y0).clone()
    ab.linear(d(g), d(W), transpose_w=True, y=acc, accumulate=True)
    torch.cuda.synchronize()

    def rel(a, b):
        return float(np.abs(a.double().cpu().numpy() - b).max() / np.abs(b).max())
    assert rel(y, f8(x) @ f8(W).T) <= 1e-5
    assert rel(gx, f8(g) @ f8(W)) <= 1e-5
    assert rel(acc, f8(y0) + f8(g) @ f8(W)) <= 1e-5


@pytest.mark.parametrize("n,compact", [(64, True), (64, False), (32, True)])
def test_latent_update_forward_and_vjp(n, compact):
    """allegro_latent_forward / _backward (reading A19) against the oracle's latent_update and its autograd VJP.  fp32, n = 64 with the
    compact scalar channel runs the tcgen05 kernels (tclin.cu: hi / lo tf32 split, TMEM accumulator), the other shapes the FMA tiles;
    333 edges = two full 128-edge tiles and a ragged one"""
    import torch

    import paper_2504_16068_b200 as ab
    from oracle import model2
    from workloads import configs, rng
    g = configs.geometry_for("C1s")
    E, rc = 333, float(g["spec"]["rc"])
    rvec = g["rvec"][:E].astype(np.float32)
    S = rng.STREAMS
    x = rng.normal(51, S["V"], (E, n)).astype(np.float32)
    sc = rng.normal(52, S["G"], (E, n)).astype(np.float32)
    A = (rng.normal(53, S["W_p"], (n, 2 * n)) / np.sqrt(2 * n)).astype(np.float32)
    gx = rng.normal(54, S["q"], (E, n)).astype(np.float32)
    gs0 = rng.normal(55, S["G"], (E, n)).astype(np.float32)          # the scalar cotangent and g_rvec are accumulated into
    gr0 = rng.normal(56, S["V"], (E, 3)).astype(np.float32)
    # oracle: float64, the VJP by autograd of <g_xnew, x_new>
    t64 = lambda a, grad=False: torch.tensor(a.astype(np.float64), requires_grad=grad)
    xo, so, ro = t64(x, True), t64(sc, True), t64(rvec, True)
    r = torch.sqrt((ro * ro).sum(1)) / rc
    u = 1.0 - 28.0 * r ** 6 + 48.0 * r ** 7 - 21.0 * r ** 8
    z_ref, xn_ref = model2.latent_update(xo, so, t64(A), u)
    (xn_ref * t64(gx)).sum().backward()
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    dV = 1 if compact else 18
    V = torch.zeros((E, n, dV), device="cuda")
    V[:, :, 0] = d(sc)
    z, xn = ab.latent_forward(d(rvec), rc, d(x), V, d(A))
    gV = torch.zeros((E, n, dV), device="cuda")
    gV[:, :, 0] = d(gs0)
    g_r = d(gr0).clone()
    g_x = ab.latent_backward(d(rvec), rc, z, d(gx), d(A), gV, g_r)
    torch.cuda.synchronize()
    tol = 1e-5

    def rel(a, b):
        b = np.asarray(b, dtype=np.float64)
        return float(np.abs(a.double().cpu().numpy() - b).max() / np.abs(b).max())
    assert rel(z, z_ref.detach().numpy()) <= tol and rel(xn, xn_ref.detach().numpy()) <= tol
    assert rel(g_x, xo.grad.numpy()) <= tol
    assert rel(gV[:, :, 0] - d(gs0), so.grad.numpy()) <= 2 * tol
    assert rel(g_r - d(gr0), ro.grad.numpy()) <= 4 * tol
    if dV > 1:
        assert float(gV[:, :, 1:].abs().max()) == 0.0


@pytest.mark.parametrize("name", ["C0", "C4s"])
def test_check_graph_accepts_sound_lists_and_names_broken_ones(name):
    """allegro_check_graph (debugging aid: the kernels index unchecked and compute-sanitizer is closed on this pool): the seeded
    graphs and their segment plans pass; one corrupted entry in each list is counted and named"""
    import torch

    import paper_2504_16068_b200 as ab
    from workloads import configs
    g = configs.geometry_for(name)
    dt = np.float64 if g["spec"]["dtype"] == "f64" else np.float32
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    rp, rev, col, rvec = d(g["row_ptr"]), d(g["rev"]), d(g["col"]), d(g["rvec"].astype(dt))
    E, N = g["rvec"].shape[0], g["row_ptr"].shape[0] - 1
    items = d(ab.segments_build(g["row_ptr"], 7))
    assert ab.check_graph(rp, E, items=items, rev=rev, col=col, rvec=rvec) == 0
    assert ab.check_graph(rp, E) == 0

    def bad(match, **kw):
        args = dict(items=items, rev=rev, col=col, rvec=rvec)
        args.update(kw)
        with pytest.raises(ab.AllegroError) as ei:
            ab.check_graph(args.pop("rp", rp), args.pop("E", E), **args)
        assert ei.value.status == 1 and match in str(ei.value), str(ei.value)

    c = int(np.argmax(np.diff(g["row_ptr"])))                 # a centre with edges
    e = int(g["row_ptr"][c])
    rp2 = rp.clone(); rp2[c + 1] = rp2[c] - 1 if c > 0 else -1
    bad("row_ptr", rp=rp2)
    bad("row_ptr", E=E + 1)
    it2 = items.clone(); it2[3, 2] += 1                        # an item reaching past its tile: the next one no longer continues it
    bad("items", items=it2)
    it3 = items[:-1].contiguous()                              # the last centre's last item is missing
    bad("items", items=it3)
    rev2 = rev.clone(); rev2[e] = rev[e + 1]                   # not an involution any more
    bad("rev", rev=rev2)
    rev3 = rev.clone(); rev3[e] = E                            # out of range
    bad("rev", rev=rev3)
    col2 = col.clone(); col2[e] = (int(col[e]) + 1) % N        # the reverse edge is not in the named neighbour's row
    bad("rev / col", col=col2)
    rv2 = rvec.clone(); rv2[e] = 0                             # zero-length edge: the kernels divide by |r|
    bad("rvec", rvec=rv2)
    rv3 = rvec.clone(); rv3[E - 1, 1] = float("nan")
    bad("rvec", rvec=rv3)
    assert ab.check_graph(rp, E, items=items, rev=rev, col=col, rvec=rvec) == 0      # the counters are reset by every call


@pytest.mark.parametrize("name", ["C0", "C1s", "C3s", "C4s"])
def test_tp_double_backward(name):
    """allegro_tp_double_backward (training, row f2; reading A26) against the oracle's term-by-term second derivative on every
    single-layer config shape (fp64 l_max 1, fp32 l_max 2 / 3)"""
    import oracle as orc
    import torch

    import paper_2504_16068_b200 as ab
    from workloads import rng
    inp = _chain.make_inputs(name)
    lmax, n, dt, rp = inp["lmax"], inp["n"], inp["dt"], inp["row_ptr"]
    E, N = inp["E"], inp["N"]
    dV, dE = 2 * (lmax + 1) ** 2, (lmax + 1) ** 2
    S = rng.STREAMS
    V, pw = inp["V"], inp["path_w"]
    G = rng.normal(21, S["G"], (E, n, dV)).astype(dt)
    aV = rng.normal(22, S["V"], (E, n, dV)).astype(dt)
    Ee = (rng.normal(23, S["W_w"], (N, n, dE)) * 0.5).astype(dt)
    bE = (rng.normal(24, S["W_w"], (N, n, dE)) * 0.5).astype(dt)
    f8 = lambda a: np.asarray(a, dtype=np.float64)
    ref = dict(zip(("dG", "dV", "dE", "dw"), orc.tp_double_backward(lmax, rp, f8(G), f8(V), f8(Ee), f8(pw), f8(aV), f8(bE))))
    plan = ab.Plan(lmax, n, ab.F64 if dt == np.float64 else ab.F32)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    got = dict(zip(("dG", "dV", "dE", "dw"), ab.tp_double_backward(plan, d(rp), d(G), d(V), d(Ee), d(pw), d(aV), d(bE))))
    torch.cuda.synchronize()
    _assert_close(ref, got, dt, keys=("dG", "dV", "dE", "dw"), label="double backward " + name)


def test_per_edge_type_cutoffs():
    """PAPER.md:156 per-edge-type cutoff radii (reading A27): the GPU neighbour builder with a species table gives the host builder's
    list and per-edge cutoffs bit for bit; the fused geometry kernels with a cutoff per edge (allegro_env_radial_forward_typed /
    _backward_typed, factorised and un-factorised forms) match the oracle's radial_typed -> env_embed chain and its VJP"""
    import oracle as orc
    import torch

    import paper_2504_16068_b200 as ab
    from workloads import configs, geometry, rng
    g = configs.geometry_for("C1s")
    pos, box, species = g["pos"], g["box"], g["species"].astype(np.int32)
    S = int(species.max()) + 1
    tab = 4.0 + 2.0 * rng.uniform(0, rng.STREAMS["rot"], np.arange(S * S)).reshape(S, S)
    tab = np.maximum(tab, tab.T)
    tab[0, 0] = 6.0
    ref = geometry.neighbour_list_periodic_typed(pos, box, species, tab)
    dt = np.float32
    nl = ab.neighbour_list(torch.from_numpy(pos).cuda(), 6.0, box=box, dtype=ab.F32, species=torch.from_numpy(species).cuda(),
                           rc_table=torch.from_numpy(np.ascontiguousarray(tab)).cuda())
    torch.cuda.synchronize()
    for k in ("row_ptr", "col", "rev"):
        assert np.array_equal(nl[k].cpu().numpy(), ref[k]), k
    assert np.array_equal(nl["rvec"].cpu().numpy(), ref["rvec"].astype(dt))
    assert np.array_equal(nl["rc_edge"].cpu().numpy(), ref["rc_edge"].astype(dt))
    assert ref["row_ptr"][-1] < g["row_ptr"][-1]          # fewer edges than with the single 6 A cutoff
    # geometry pass with per-edge cutoffs
    lmax, n = 2, 64
    rp, rvec, rce = ref["row_ptr"], ref["rvec"].astype(dt), ref["rc_edge"].astype(dt)
    N = rp.shape[0] - 1
    Wr = (rng.normal(3, rng.STREAMS["W_r"], (n, 8)) / np.sqrt(8)).astype(dt)
    gE = rng.normal(3, rng.STREAMS["G"], (N, n, 9)).astype(dt)
    f8 = lambda a: np.asarray(a, dtype=np.float64)
    w, dwdr = orc.radial_typed(f8(Wr), f8(rce), f8(rvec))
    Eenv = orc.env_embed(lmax, rp, f8(rvec), w, 0.7)
    g_r, g_w = orc.env_embed_backward(lmax, rp, f8(gE), f8(rvec), w, 0.7)
    orc.radial_backward(f8(rvec), g_w, dwdr, g_r)
    plan = ab.Plan(lmax, n, ab.F32)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    for want in (False, True):          # factorised form; un-factorised form (w / g_w requested)
        E2, w2 = ab.env_radial_forward_typed(plan, d(rp), d(rvec), d(Wr), d(rce), 0.7, want_w=want)
        gr2, gw2 = ab.env_radial_backward_typed(plan, d(rp), d(gE), d(rvec), d(Wr), d(rce), 0.7, want_g_w=want)
        torch.cuda.synchronize()
        _assert_close(dict(Eenv=Eenv, w=w, g_r=g_r, g_w=g_w), dict(Eenv=E2, w=w2, g_r=gr2, g_w=gw2), dt, keys=("Eenv", "w", "g_r", "g_w"),
                      label="typed cutoffs want_w=%s" % want)


@pytest.mark.parametrize("geom,lmax,n,n_in,dt", [("C1s", 2, 64, 64, np.float32), ("C0", 1, 8, 12, np.float64), ("C4s", 3, 32, 64, np.float32)])
def test_env_linear_forward_and_vjp(geom, lmax, n, n_in, dt):
    """allegro_env_linear_forward / _backward (embedding of the linear weights w = x W^T with the linear map applied once per centre)
    against the oracle's plain chain: w = x W^T -> env_embed; VJP: env_embed_backward -> g_x = g_w W; also accumulating"""
    import oracle as orc
    import torch

    import paper_2504_16068_b200 as ab
    from workloads import configs, rng
    g = configs.geometry_for(geom)
    rp, rvec = g["row_ptr"], g["rvec"].astype(dt)
    E, N = rvec.shape[0], rp.shape[0] - 1
    dE = (lmax + 1) ** 2
    S = rng.STREAMS
    x = rng.normal(17, S["V"], (E, n_in)).astype(dt)
    W = (rng.normal(17, S["W_w"], (n, n_in)) / np.sqrt(n_in)).astype(dt)
    gE = rng.normal(17, S["G"], (N, n, dE)).astype(dt)
    f8 = lambda a: np.asarray(a, dtype=np.float64)
    w = f8(x) @ f8(W).T
    Eenv = orc.env_embed(lmax, rp, f8(rvec), w, 0.8)
    g_r, g_w = orc.env_embed_backward(lmax, rp, f8(gE), f8(rvec), w, 0.8)
    g_x = g_w @ f8(W)
    plan = ab.Plan(lmax, n, ab.F64 if dt == np.float64 else ab.F32)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    rpd, rd, xd, Wd, gEd = d(rp), d(rvec), d(x), d(W), d(gE)
    E2 = ab.env_linear_forward(plan, rpd, rd, xd, Wd, 0.8)
    gr2, gx2 = ab.env_linear_backward(plan, rpd, gEd, rd, xd, Wd, 0.8, torch.empty_like(rd), torch.empty_like(xd))
    torch.cuda.synchronize()
    _assert_close(dict(Eenv=Eenv, g_r=g_r, g_x=g_x), dict(Eenv=E2, g_r=gr2, g_x=gx2), dt, keys=("Eenv", "g_r", "g_x"), label="env_linear " + geom)
    gr3, gx3 = torch.ones_like(rd), torch.ones_like(xd)
    ab.env_linear_backward(plan, rpd, gEd, rd, xd, Wd, 0.8, gr3, gx3, accumulate_g_rvec=True, accumulate_g_x=True)
    _assert_close(dict(g_r=g_r + 1.0, g_x=g_x + 1.0), dict(g_r=gr3, g_x=gx3), dt, keys=("g_r", "g_x"), label="env_linear accumulate " + geom)


def test_layer1_outer_product_input():
    """allegro_tp_forward_outer / _backward_outer / allegro_edge_embed_factors(_backward): the first layer with its input
    V0 = v0 (x) Y(rhat) generated on chip equals the same layer fed with the materialised V0 (allegro_edge_embed -> allegro_tp_forward /
    _backward), and the contracted cotangents g_v0, gY equal the contractions of that path's gV with the ORACLE's Y_lm; then the
    embedding's VJP from the factors equals the one from gV0"""
    import oracle as orc
    import torch

    import paper_2504_16068_b200 as ab
    from workloads import configs, rng
    lmax, n, dt = 2, 64, np.float32
    g = configs.geometry_for("C1s")
    rp, rvec = g["row_ptr"], g["rvec"].astype(dt)
    E, N = rvec.shape[0], rp.shape[0] - 1
    S = rng.STREAMS
    W_x0 = (rng.normal(19, S["W_x0"], (n, 8)) / np.sqrt(8)).astype(dt)
    W_v0 = (rng.normal(19, S["W_v0"], (n, 8)) / np.sqrt(8)).astype(dt)
    Ee = (rng.normal(19, S["W_w"], (N, n, 9)) * 0.5).astype(dt)
    W = (rng.normal(19, S["W_p"], (30, n, n)) / np.sqrt(n)).astype(dt)
    G = rng.normal(19, S["G"], (E, n, 18)).astype(dt)
    gs = rng.normal(20, S["q"], (E, n, 1)).astype(dt)
    g_x0 = rng.normal(21, S["q"], (E, n)).astype(dt)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    rpd, rd, Ed, Wd, Gd, gsd, Wx, Wv, gx0 = d(rp), d(rvec), d(Ee), d(W), d(G), d(gs), d(W_x0), d(W_v0), d(g_x0)
    plan = ab.Plan(lmax, n, ab.F32, ab.W_DENSE)
    plan.set_in_blocks(0x19)
    rc = 6.0
    # materialised path
    x0, V0 = ab.edge_embed(plan, rd, Wx, Wv, rc)
    out_a, sc_a = torch.empty_like(V0), torch.empty((E, n, 1), dtype=V0.dtype, device="cuda")
    ab.tp_forward_aux(plan, rpd, V0, Ed, Wd, out_a, sc_a)
    gV_a, gE_a = ab.tp_backward_aux(plan, rpd, Gd, gsd, V0, Ed, Wd, torch.empty_like(V0), torch.empty_like(Ed))
    gr_a = torch.zeros_like(rd)
    ab.edge_embed_backward(plan, rd, Wx, Wv, rc, gx0, gV_a, gr_a)
    # on-chip path
    x0b, v0 = ab.edge_embed_factors(plan, rd, Wx, Wv, rc, torch.empty_like(x0), torch.empty_like(x0))
    assert torch.equal(x0b, x0)
    out_b, sc_b = torch.empty_like(V0), torch.empty_like(sc_a)
    ab.tp_forward_outer(plan, rpd, rd, v0, Ed, Wd, out_b, sc_b)
    g_v0, gY, gE_b = ab.tp_backward_outer(plan, rpd, Gd, gsd, rd, v0, Ed, Wd, torch.empty_like(x0), torch.empty((E, 9), dtype=V0.dtype, device="cuda"),
                                          torch.empty_like(Ed))
    gr_b = torch.zeros_like(rd)
    ab.edge_embed_factors_backward(plan, rd, Wx, Wv, rc, gx0, g_v0, gY, gr_b)
    torch.cuda.synchronize()
    Y = np.stack([orc.sph_harm(lmax, rvec[e].astype(np.float64))[0] for e in range(E)])
    slots = [0, 5, 6, 7, 8, 9, 10, 11, 12]
    gVn = gV_a.double().cpu().numpy()[:, :, slots]
    ref = dict(out=out_a, sc=sc_a, gEenv=gE_a, g_r=gr_a, g_v0=np.einsum("enj,ej->en", gVn, Y),
               gY=np.einsum("enj,en->ej", gVn, v0.double().cpu().numpy()))
    ref = {k: (v.double().cpu().numpy() if hasattr(v, "cpu") else v) for k, v in ref.items()}
    got = dict(out=out_b, sc=sc_b, gEenv=gE_b, g_r=gr_b, g_v0=g_v0, gY=gY)
    _assert_close(ref, got, dt, keys=tuple(ref.keys()), label="layer-1 outer")

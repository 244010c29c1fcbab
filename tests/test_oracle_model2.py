"""Pins of the two-layer model oracle (oracle/model2.py, reading A19): nothing here compares it with the CUDA path."""
import numpy as np
import pytest
import torch

import oracle as orc
from oracle import model2
from workloads.inputs import make_model_inputs


@pytest.fixture(scope="module")
def small():
    inp = make_model_inputs("C0", n=4, lmax=2, n_layers=2)
    inp["rvec"] = inp["rvec"].astype(np.float64)
    return inp


def test_sph_harm_torch_matches_cpp_oracle():
    rng_ = np.random.default_rng(1)
    r = rng_.normal(size=(20, 3))
    u = r / np.linalg.norm(r, axis=1, keepdims=True)
    for lmax in (1, 2, 3):
        Yt = model2.sph_harm_torch(lmax, torch.from_numpy(u)).numpy()
        Yc = np.stack([orc.sph_harm(lmax, u[i])[0] for i in range(u.shape[0])])
        assert np.max(np.abs(Yt - Yc)) < 1e-13
        for l in range(lmax + 1):      # component normalisation: sum_m Y_lm^2 = 2l+1
            assert np.allclose((Yt[:, l * l:(l + 1) ** 2] ** 2).sum(1), 2 * l + 1, atol=1e-12)


def test_gradient_vs_central_differences(small):
    p, rp, rvec = small["params"], small["row_ptr"], small["rvec"]
    en, g = model2.energy_grad(p, rp, rvec)
    rng_ = np.random.default_rng(0)
    h = 1e-5
    for _ in range(8):
        e, d = int(rng_.integers(rvec.shape[0])), int(rng_.integers(3))
        rp_, rm_ = rvec.copy(), rvec.copy()
        rp_[e, d] += h
        rm_[e, d] -= h
        fd = (float(model2.forward(p, rp, torch.from_numpy(rp_))) - float(model2.forward(p, rp, torch.from_numpy(rm_)))) / (2 * h)
        assert abs(fd - g[e, d]) <= 1e-6 * max(1.0, np.abs(g).max()), (e, d, fd, g[e, d])


@pytest.mark.parametrize("improper", [False, True])
def test_energy_invariant_under_rotation_and_inversion(small, improper):
    p, rp, rvec = small["params"], small["row_ptr"], small["rvec"]
    R = orc.rotation_matrix(0.7, 1.1, -0.4)
    if improper:
        R = -R
    e0, g0 = model2.energy_grad(p, rp, rvec)
    e1, g1 = model2.energy_grad(p, rp, rvec @ R.T)
    assert abs(e0 - e1) <= 1e-10 * max(1.0, abs(e0))
    assert np.max(np.abs(g1 - g0 @ R.T)) <= 1e-9 * np.abs(g0).max()      # the gradient is a vector (covariant)


def test_layers_match_cpp_oracle_primitives_and_forces_sum_to_zero(small):
    p, rp, rvec = small["params"], small["row_ptr"], small["rvec"]
    taps = []
    en, g = model2.energy_grad(p, rp, rvec, taps)
    for layer in range(p["n_layers"]):
        t = taps[layer]
        Eenv = orc.env_embed(p["lmax"], rp, rvec, t["w"], p["scale"])
        assert np.max(np.abs(Eenv - t["Eenv"])) <= 1e-12 * np.abs(Eenv).max()
        out = orc.tp_forward(p["lmax"], rp, t["V_in"], Eenv, p["W_p"][layer])
        assert np.max(np.abs(out - t["V_out"])) <= 1e-12 * np.abs(out).max()
    # layer-1 input features occupy the natural-parity slots only (reading A19)
    V0 = taps[0]["V_in"]
    for l in range(p["lmax"] + 1):
        o = model2.feature_offset(l, l % 2 == 0)      # the other parity
        assert np.all(V0[:, :, o:o + 2 * l + 1] == 0.0)
    assert abs(en - taps[-1]["e_edge"].sum()) <= 1e-12 * abs(en)
    F = orc.force_gather(rp, small["rev"], g)
    assert np.abs(F.sum(0)).max() <= 1e-10 * np.abs(F).max()

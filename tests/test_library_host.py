"""CPU-side checks of the product library (no GPU): the shared library loads and exports every symbol of
include/allegro_b200.h, the host plan builder (ladder-operator CG) equals the oracle's tables (integers
bit-exact, coefficients to 1e-14: SURVEY 8.a8), the segment plan equals the oracle's, argument checks
return status codes, and the product package shares no code with oracle/."""
import os
import re

import numpy as np
import pytest

import oracle as orc
import paper_2504_16068_b200 as ab

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "allegro_b200.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(allegro_[a-z0-9_]+)\s*\(", hdr))
    assert len(declared) >= 20
    L = ab.lib()
    for name in sorted(declared):
        assert hasattr(L, name), "library does not export " + name
    assert declared == set(ab.SIGNATURES), "binding and header disagree: %s" % (declared ^ set(ab.SIGNATURES))


@pytest.mark.parametrize("lmax", [1, 2, 3])
def test_plan_tables_equal_oracle(lmax):
    plan = ab.Plan(lmax, 8, ab.F64, ab.W_SCALAR)
    assert plan.dV == orc.dim_v(lmax) and plan.dE == orc.dim_e(lmax)
    po, pl = orc.paths(lmax), plan.paths()
    assert plan.P == len(po["l1"])
    for k in po:
        assert np.array_equal(po[k], pl[k]), k
    co, cl = orc.cg_list(lmax), plan.cg()
    assert plan.nnz == len(co["coef"]) == {1: 32, 2: 274, 3: 1222}[lmax]
    for k in ("path", "i", "j", "k"):
        assert np.array_equal(co[k], cl[k]), k
    assert np.max(np.abs(co["coef"] - cl["coef"])) < 1e-14


def test_cg_real_block_ladder_vs_racah():
    for l1 in range(4):
        for l2 in range(4):
            for l3 in range(abs(l1 - l2), min(l1 + l2, 3) + 1):
                a = ab.cg_real_block(l1, l2, l3)
                b, _, _ = orc.cg_real(l1, l2, l3)
                assert np.max(np.abs(a - b)) < 1e-14, (l1, l2, l3)


def test_segment_plan_equals_oracle():
    rng = np.random.default_rng(0)
    for T in (1, 3, 16, 128):
        deg = rng.integers(0, 40, size=50)
        deg[[3, 17]] = 0
        rp = np.concatenate([[0], np.cumsum(deg)]).astype(np.int32)
        assert np.array_equal(ab.segments_build(rp, T), orc.segments(rp, T))


def test_status_codes_without_gpu():
    import ctypes as C
    L = ab.lib()
    h = C.c_void_p()
    assert L.allegro_plan_create(7, 0, 8, 0, 0, C.byref(h)) == 2          # EUNSUPPORTED
    assert b"unsupported" in L.allegro_last_error()
    assert L.allegro_plan_create(2, 0, 0, 0, 0, C.byref(h)) == 1          # EINVAL
    assert L.allegro_plan_create(2, 0, 8, 5, 0, C.byref(h)) == 1
    assert L.allegro_status_str(3) == b"ALLEGRO_ECUDA"
    plan = ab.Plan(2, 64)
    # NULL tensors with non-zero sizes are rejected before any CUDA call
    assert L.allegro_tp_forward(plan.h, 4, 10, None, None, 0, None, None, None, None, None) == 1
    assert L.allegro_env_embed(plan.h, 4, 10, None, None, 0, None, None, 1.0, None, None, 0, None) == 1
    assert L.allegro_launch_count() == 0


def test_product_and_oracle_share_no_code():
    """neither side includes / imports the other"""
    def code_lines(path):
        return [ln for ln in open(path, errors="ignore").read().splitlines()
                if re.match(r"\s*(#\s*include|import |from )", ln) or "CDLL" in ln or "dlopen" in ln]

    pkg = os.path.join(ROOT, "paper_2504_16068_b200")
    for dirpath, _, files in os.walk(pkg):
        if "build" in dirpath.split(os.sep):
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                for ln in code_lines(os.path.join(dirpath, f)):
                    assert "oracle" not in ln, (f, ln)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            for ln in code_lines(os.path.join(ROOT, "oracle", f)):
                assert "allegro_b200" not in ln and "paper_2504_16068_b200" not in ln and "plan.h" not in ln, (f, ln)

"""The C-ABI library loads and exports every symbol include/*.h declares; argument validation that needs no
GPU (status codes, workspace sizing).  No compute calls here."""
import ctypes as C
import os
import re

import pytest

from paper_2105_08026_b200 import binding as B
from paper_2105_08026_b200 import build as cuda_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    cuda_build.build()
    return B.load()


def declared_symbols():
    names = set()
    inc = os.path.join(ROOT, "include")
    for f in sorted(os.listdir(inc)):
        src = open(os.path.join(inc, f)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(cudahm_[a-z0-9_]+)\s*\(", src))
    return sorted(names)


def test_every_declared_symbol_is_exported(lib):
    decl = declared_symbols()
    assert len(decl) >= 18
    for name in decl:
        assert hasattr(lib, name), f"{name} is declared in include/ but not exported by libcudahm.so"
    assert sorted(B.EXPORTS) == decl, "binding.EXPORTS must list exactly the declared entry points"


def test_model_dims_and_workspace(lib):
    assert B.model_dims(B.M_NORMAL1D) == dict(p=1, dtheta=2, n_cols=2, n_consts=0)
    assert B.model_dims(B.M_THINNED_SCHECHTER1D) == dict(p=1, dtheta=3, n_cols=2, n_consts=6)
    assert B.model_dims(B.M_BINORMAL2D) == dict(p=2, dtheta=5, n_cols=4, n_consts=0)
    assert B.model_dims(B.M_LINREG_ME1D) == dict(p=1, dtheta=3, n_cols=3, n_consts=0)
    assert B.model_dims(B.M_BB1_FLUXNOISE1D) == dict(p=1, dtheta=3, n_cols=2, n_consts=7)
    assert B.model_dims(B.M_NORMAL3D_KNOWNCOV) == dict(p=3, dtheta=3, n_cols=3, n_consts=9)
    with pytest.raises(B.CudahmError):
        B.model_dims(99)
    small = B.workspace_bytes(B.make_config(B.M_BINORMAL2D, 1000))
    big = B.workspace_bytes(B.make_config(B.M_BINORMAL2D, 1_000_000))
    # chi 2 + L 3 + data 4 columns of 8 bytes
    assert big - small >= (1_000_000 - 1024) * 9 * 8
    with_mom = B.workspace_bytes(B.make_config(B.M_BINORMAL2D, 1_000_000, keep_chi_moments=True))
    assert with_mom - big >= 1_000_000 * 2 * 8 * 3
    f32 = B.workspace_bytes(B.make_config(B.M_LINREG_ME1D, 10_000_000, precision=B.F32_STATE_F64_REDUCE))
    assert 10_000_000 * 5 * 4 <= f32 <= 10_000_000 * 5 * 4 + (16 << 20)   # + mailboxes, slots, tables


def test_invalid_configs_are_refused(lib):
    bad = B.make_config(B.M_NORMAL1D, 10)
    bad.p = 2
    assert B.workspace_bytes(bad) == 0
    bad = B.make_config(B.M_NORMAL1D, 10)
    bad.struct_size = 8
    assert B.workspace_bytes(bad) == 0
    bad = B.make_config(B.M_NORMAL1D, 10, target_accept_chi=1.5)
    assert B.workspace_bytes(bad) == 0
    bad = B.make_config(B.M_NORMAL1D, 10, block_threads=100)
    assert B.workspace_bytes(bad) == 0
    # sharding: the offset must be even (objects draw in pairs) and the shard must lie inside the population
    assert B.workspace_bytes(B.make_config(B.M_NORMAL1D, 10, object_offset=3, n_objects_total=100)) == 0
    assert B.workspace_bytes(B.make_config(B.M_NORMAL1D, 10, object_offset=96, n_objects_total=100)) == 0
    assert B.workspace_bytes(B.make_config(B.M_NORMAL1D, 10, object_offset=90, n_objects_total=100)) > 0
    # hooks: a negative prior precision or a negative freeze iteration is refused
    assert B.workspace_bytes(B.make_config(B.M_NORMAL1D, 10, prior_mean=[0.0, 0.0], prior_sd=[-1.0, 1.0])) == 0
    assert B.workspace_bytes(B.make_config(B.M_NORMAL1D, 10, adapt_until=-1)) == 0
    # flags: the documented bits (streaming only, TMA staging, prefetch on / off, staged draw steps) pass; others do not
    ok = B.FLAG_STREAMING_ONLY | B.FLAG_PREFETCH_ON | B.flag_stage_steps(3)
    assert B.workspace_bytes(B.make_config(B.M_NORMAL1D, 10, flags=ok)) > 0
    assert B.workspace_bytes(B.make_config(B.M_NORMAL1D, 10, flags=B.flag_stage_steps(0) | B.FLAG_PREFETCH_OFF)) > 0
    assert B.workspace_bytes(B.make_config(B.M_NORMAL1D, 10, flags=1 << 16)) == 0
    assert B.workspace_bytes(B.make_config(B.M_NORMAL1D, 10, flags=1 << 20)) == 0
    assert B.flag_stage_steps(0) == 0x100 and B.flag_stage_steps(2) == 0x300
    cfg = B.make_config(B.M_NORMAL3D_KNOWNCOV, 10, precision=B.F32_STATE_F64_REDUCE)
    h = C.c_void_p()
    assert lib.cudahm_create(C.byref(cfg), None, 0, None, C.byref(h)) == B.E_UNSUPPORTED
    assert lib.cudahm_shard_sweep(None, 0, 1, None) == B.E_INVALID
    h = C.c_void_p()
    cfg = B.make_config(B.M_NORMAL1D, 10)
    assert lib.cudahm_create(C.byref(cfg), None, 0, None, C.byref(h)) == B.E_WORKSPACE
    assert b"workspace" in lib.cudahm_last_error(None)
    cfg = B.make_config(B.M_BINORMAL2D, 10, precision=B.F32_STATE_F64_REDUCE)
    assert lib.cudahm_create(C.byref(cfg), None, 0, None, C.byref(h)) == B.E_UNSUPPORTED
    assert lib.cudahm_run(None, 1, 0, 1) == B.E_INVALID
    assert lib.cudahm_sync(None) == B.E_INVALID


def test_no_oracle_in_product_path():
    """The package never imports, links or executes anything under oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_2105_08026_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle|#include\s+\"(\.\./)*oracle", src, flags=re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".hpp", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2105_08026_b200" not in src.replace("paper_2105_08026_b200/csrc (the CUDA path)", ""), f
            assert "cuda_runtime" not in src, f

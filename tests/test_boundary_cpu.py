"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol that
include/rmsynth.h declares, validates arguments before touching the device, and fails
loudly (no CPU fallback) when no B200 is present."""
import ctypes
import os
import re

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def b():
    from paper_1810_06250_b200 import build
    build.build()
    from paper_1810_06250_b200 import binding
    return binding


def test_every_declared_symbol_is_exported(b):
    hdr = open(os.path.join(ROOT, "include", "rmsynth.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(rmsynth_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(b.EXPORTS)
    lib = ctypes.CDLL(b.LIB_PATH)
    for name in declared:
        assert getattr(lib, name) is not None


def test_version_and_strerror(b):
    assert "sm_100a" in b.rmsynth_version()
    assert b._lib.rmsynth_strerror(b.EINVAL) == b"invalid argument"


@pytest.mark.parametrize("kw", [
    dict(nu=[1e9, -1.0]), dict(nu=[1e9, np.inf]), dict(w=[1.0, -0.5]), dict(w=[0.0, 0.0]),
    dict(phi=[np.nan]), dict(scheme=5), dict(scheme=99), dict(lambda0_mode=7), dict(nu=[], w=None),
    dict(phi=[]),
])
def test_plan_create_rejects_bad_arguments_before_touching_the_device(b, kw):
    a = dict(nu=[1e9, 1.1e9], w=[1.0, 1.0], phi=[0.0, 1.0], scheme=b.SCHEME_FP32_TABLE, lambda0_mode=0)
    a.update(kw)
    with pytest.raises(b.RmsynthError) as e:
        b.Plan(a["nu"], a["w"], a["phi"], scheme=a["scheme"], lambda0_mode=a["lambda0_mode"])
    assert e.value.status == b.EINVAL


def test_no_gpu_means_loud_failure_not_fallback(b):
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(b.RmsynthError) as e:
        b.Plan([1e9, 1.1e9], None, [0.0, 1.0])
    assert e.value.status in (b.ECUDA, b.EUNSUPPORTED)


def test_null_plan_is_einval(b):
    assert b._lib.rmsynth_execute(None, None, None, 4, 0, None, None, None) == b.EINVAL
    assert b._lib.rmsynth_plan_destroy(None) == b.OK
    assert b._lib.rmsynth_rmsf(None, None, 0, None, None) == b.EINVAL


def test_product_path_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1810_06250_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.lower(), f"{f} mentions the oracle"


def test_committed_ncu_evidence_belongs_to_the_committed_tensor_sources():
    """bench.py quotes `traffic` and the tensor-pipe activity from profiles/r03_ncu_summary.json only when that capture was
    taken with the tensor-path sources that run; a kernel edit without a new capture must not go unnoticed."""
    import importlib.util
    import json
    spec = importlib.util.spec_from_file_location("bench_module", os.path.join(ROOT, "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    with open(os.path.join(ROOT, "profiles", "r03_ncu_summary.json")) as f:
        captures = json.load(f)["captures"]
    assert "5:f16x3" in captures
    for key, e in captures.items():
        assert e["tensor_path_hash"] == bench.tensor_path_hash(), f"{key}: re-capture with ncu (profiles/r03_ncu_kernels.md names the commands)"
        assert e["dram_bytes"] > 0 and 0 < e["tensor_pipe_elapsed_pct"] <= e["tensor_pipe_active_pct"] <= 100
    assert bench.ncu_evidence(5, "f16x3") is not None

"""The C-ABI library loads on a CPU-only box and exports every symbol that
include/monc_adv.h declares; argument validation happens before any CUDA call.
No compute is attempted here."""
import ctypes as C
import os
import re

import pytest

from paper_2009_12850_b200 import binding
from paper_2009_12850_b200 import build as libbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "monc_adv.h")
TUNING_HEADER = os.path.join(ROOT, "include", "monc_adv_tuning.h")  # internal knobs, same library


@pytest.fixture(scope="module")
def lib():
    libbuild.build()
    return binding.load()


def declared_functions(headers=(HEADER, TUNING_HEADER)):
    names = set()
    for path in headers:
        src = re.sub(r"/\*.*?\*/", "", open(path).read(), flags=re.S)
        names |= set(re.findall(r"\b(monc_adv_[a-z_0-9]+)\s*\(", src))
    return sorted(names)


def test_header_symbols_all_exported(lib):
    names = declared_functions()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/ but not exported"
    assert sorted(binding.SYMBOLS) == names, "binding.SYMBOLS out of sync with the headers"
    # the kernel-geometry knobs live in the internal header only
    public = declared_functions((HEADER,))
    for n in ("monc_adv_set_tuning", "monc_adv_set_variant", "monc_adv_set_pdl", "monc_adv_set_cluster", "monc_adv_set_l2_hint", "monc_adv_plan_describe", "monc_adv_set_graph", "monc_adv_graph_state"):
        assert n not in public and n in names


def test_version_string(lib):
    assert "sm_100a" in binding.version()


def test_create_validates_before_cuda(lib):
    import numpy as np
    from paper_2009_12850_b200 import synth
    g = synth.grid(8)
    bad = [
        dict(nx=0, ny=4, nz=8, halo=2), dict(nx=4, ny=4, nz=2, halo=2),
        dict(nx=4, ny=4, nz=8, halo=0),
    ]
    for kw in bad:
        with pytest.raises(binding.MoncAdvError) as e:
            binding.MoncAdv(dx=50.0, dy=50.0, dz=g["dz"], dzn=g["dzn"], rho=g["rho"], rhon=g["rhon"], **kw)
        assert e.value.code == binding.EINVAL
    with pytest.raises(binding.MoncAdvError) as e:
        binding.MoncAdv(4, 4, 8, 2, -1.0, 50.0, g["dz"], g["dzn"], g["rho"], g["rhon"])
    assert e.value.code == binding.EINVAL
    with pytest.raises(binding.MoncAdvError) as e:  # only some tz arrays given
        binding.MoncAdv(4, 4, 8, 2, 50.0, 50.0, g["dz"], g["dzn"], g["rho"], g["rhon"], tzc1=np.zeros(8))
    assert e.value.code == binding.EINVAL
    with pytest.raises(binding.MoncAdvError) as e:
        binding.MoncAdv(4, 4, 8, 2, 50.0, 50.0, g["dz"], g["dzn"], g["rho"], g["rhon"], dtype=7)
    assert e.value.code == binding.EINVAL


def test_no_cpu_fallback_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2009_12850_b200 import synth
    g = synth.grid(8)
    with pytest.raises(binding.MoncAdvError) as e:
        binding.MoncAdv(4, 4, 8, 2, 50.0, 50.0, g["dz"], g["dzn"], g["rho"], g["rhon"])
    assert e.value.code in (binding.ECUDA, binding.ENOMEM)


def test_null_handle_calls_return_einval(lib):
    assert lib.monc_adv_set_chunks(None, 4) == binding.EINVAL
    assert lib.monc_adv_launch_count(None) == 0
    lib.monc_adv_destroy(None)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2009_12850_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "monc_adv_oracle" not in txt, f
    otxt = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + \
        open(os.path.join(ROOT, "oracle", "monc_adv_oracle.cpp")).read()
    assert "paper_2009_12850_b200" not in otxt.replace("paper_2009_12850_b200/csrc", "")


def test_plan_chunks_host_rule(lib):
    # a hybrid step takes T (1 + 1/C) + C c; the library takes the power of two nearest
    # sqrt(T / c) with T = bytes of one direction at 49.5 GB/s, c = 15 us + 5 us per copy.  Host arithmetic only.
    assert binding.plan_chunks(512, 512, 256, 2, "f64", 13, 13) == 32    # config 2: measured best 32
    assert binding.plan_chunks(1024, 1024, 160, 2, "f64", 7, 7) == 64    # config 4: 32..64 measured equal
    assert binding.plan_chunks(256, 256, 128, 2, "f64", 3, 3) == 8       # config 1's shape: measured best 8
    assert binding.plan_chunks(512, 512, 256, 2, "f32", 13, 13) == 16    # half the bytes
    assert binding.plan_chunks(16, 16, 32, 2, "f64", 3, 3) == 1          # config 0: one chunk
    assert binding.plan_chunks(3, 2048, 256, 2, "f64", 13, 13) <= 3      # never more chunks than x planes
    counts = [binding.plan_chunks(n, n, 128, 2, "f64", 5, 5) for n in (32, 64, 128, 256, 512, 1024, 2048)]
    assert counts == sorted(counts) and all(c & (c - 1) == 0 for c in counts) and counts[-1] <= 64
    with pytest.raises(binding.MoncAdvError):
        binding.plan_chunks(0, 4, 4, 2, "f64", 3, 3)

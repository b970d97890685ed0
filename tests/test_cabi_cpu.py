"""CPU-side checks of the boundary: the C-ABI library loads, exports every symbol include/nf.h declares,
validates its arguments on the host, and refuses to compute without a CUDA device (no CPU fallback)."""
import ctypes
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "nf.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(nf_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    import paper_2110_11398_b200 as nf
    lib = ctypes.CDLL(nf.LIB_PATH)
    syms = declared_symbols()
    assert {"nf_plan_create", "nf_bin", "nf_accel", "nf_destroy"} <= set(syms)
    for s in syms:
        assert hasattr(lib, s), f"{s} declared in include/nf.h but not exported"
    assert sorted(nf.EXPORTS) == syms


def test_library_is_sm100a_only():
    import subprocess
    import paper_2110_11398_b200 as nf
    out = subprocess.run(["cuobjdump", "-lelf", nf.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    assert not re.search(r"sm_(?!100a)\d+", out)


def test_plan_validation():
    import paper_2110_11398_b200 as nf
    for args in [(4, 1.0, 0.01, 2), (5, 1.0, 0.01, 5), (5, 1.0, 0.01, -1), (5, 0.0, 0.01, 2), (5, -1.0, 0.01, 2),
                 (5, 1.0, -0.1, 2), (5, float("nan"), 0.01, 2), (1626, 1.0, 0.0, 2), (5, 1.0, 1e-12, 2)]:
        with pytest.raises(nf.NFError):
            nf.nf_plan_create(*args)
        assert nf.nf_last_error()
    for args in [(5, 1.0, 0.0, 2), (1, 1.0, 0.1, 0), (251, 1.0, 1 / 40960, 2), (9, 2000.0, 25.0, 4)]:
        h = nf.nf_plan_create(*args)
        st = nf.nf_get_stats(h)
        assert st["cells"] == args[0] ** 3 and st["n"] == 0
        nf.nf_destroy(h)
    nf.nf_destroy(None)          # NULL-safe


def test_workspace_bytes_and_options():
    import paper_2110_11398_b200 as nf
    h = nf.nf_plan_create(63, 1.0, 1 / 10240, 2)
    sizes = [nf.nf_workspace_bytes(h, n) for n in (0, 1, 1000, 10 ** 6, 256 ** 3)]
    assert all(a <= b for a, b in zip(sizes, sizes[1:])) and sizes[0] > 0
    assert sizes[-1] < 60 * 256 ** 3          # < 60 B/particle
    nf.nf_set_option(h, "variant", 1)
    nf.nf_set_option(h, "heavy_first", 0)
    with pytest.raises(nf.NFError):
        nf.nf_set_option(h, "no_such_option", 1)
    with pytest.raises(nf.NFError):
        nf.nf_set_option(h, "variant", 7)
    nf.nf_destroy(h)


@pytest.mark.skipif(torch.cuda.is_available(), reason="only meaningful without a GPU")
def test_no_cpu_fallback():
    """Without a device every compute entry point fails loudly with NF_ERR_CUDA / NF_ERR_STATE."""
    import paper_2110_11398_b200 as nf
    B = nf.binding
    h = nf.nf_plan_create(5, 1.0, 0.01, 2)
    pos = torch.rand((10, 3))
    with pytest.raises(nf.NFError) as e:
        nf.nf_bin_host(h, pos)
    assert e.value.code == B.NF_ERR_CUDA and "no CPU fallback" in str(e.value)
    with pytest.raises(nf.NFError) as e:
        nf.nf_accel_host(h, torch.empty((10, 3)))
    assert e.value.code == B.NF_ERR_STATE
    nf.nf_destroy(h)


def test_product_does_not_import_oracle():
    """The product path shares nothing with the oracle (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_2110_11398_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                txt = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert "nf_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2110_11398_b200" not in txt and "from paper_2110_11398_b200" not in txt, f
            assert '#include "nf.h"' not in txt and "nf_internal" not in txt, f

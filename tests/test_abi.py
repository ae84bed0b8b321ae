"""The C-ABI library builds, loads and exports every symbol include/negf.h declares (CPU only;
no compute calls without a GPU)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "negf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(negf_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(negf_lib):
    names = _declared()
    assert len(names) >= 15
    lib = ctypes.CDLL(negf_lib.LIB_PATH)
    for nm in names:
        assert hasattr(lib, nm), f"{nm} declared in negf.h but not exported"
    assert sorted(negf_lib.EXPORTS) == names


def test_strerror_and_argument_errors(negf_lib):
    assert negf_lib.strerror(0) == "ok"
    assert "workspace" in negf_lib.strerror(negf_lib.ENOWORKSPACE)
    # argument errors are detected before any CUDA work
    assert negf_lib.lib.negf_rgf_retarded(None, None, None, None, None, None, None, 0, None) == negf_lib.EINVAL
    assert negf_lib.lib.negf_obc_decimate(None, None, None, 0, 0.0, 1.0, 1e-12, 10, *([None] * 8)) == negf_lib.EINVAL
    p = negf_lib.Problem(4, 8, 2, None, None, None, None, None, 1e-6)
    n = negf_lib.Context.workspace_bytes(p)
    assert n > 4 * 8 * 8 * 16 * 2 * 3


def test_no_cpu_fallback(negf_lib):
    """Without a compute-capability-10 GPU the context refuses to exist."""
    import torch
    if torch.cuda.is_available() and torch.cuda.get_device_capability(0)[0] == 10:
        return
    try:
        negf_lib.Context(0)
    except negf_lib.NegfError:
        return
    raise AssertionError("Context() must fail without a B200-class GPU")


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2602_03438_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2602_03438_b200" not in src.replace("`paper_2602_03438_b200/`", ""), f

"""CPU-side checks of the C-ABI boundary (no GPU, no compute calls): libdpb.so builds for sm_100a, loads, and
exports every symbol include/dpb.h declares; the Python binding refuses to run without a device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "dpb.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dpb_[a-z_0-9]+)\s*\(", text)))


@pytest.fixture(scope="module")
def lib():
    from paper_2004_11658_b200 import build
    return ctypes.CDLL(build.build())


def test_header_declares_the_contract():
    names = _declared_symbols()
    for must in ("dpb_model_create", "dpb_model_destroy", "dpb_eval", "dpb_eval_host", "dpb_build_nlist",
                 "dpb_last_error"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    for name in _declared_symbols():
        assert hasattr(lib, name), f"libdpb.so does not export {name}"


def test_version_and_error_strings(lib):
    lib.dpb_version.restype = ctypes.c_char_p
    lib.dpb_last_error.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.dpb_version()
    assert isinstance(lib.dpb_last_error(), bytes)


def test_create_rejects_bad_arguments_without_a_gpu(lib):
    """Argument validation happens before any CUDA call: EINVAL for null pointers and for precisions outside the enum."""
    out = ctypes.c_void_p()
    assert lib.dpb_model_create(None, 0, ctypes.byref(out)) == -1

    class Desc(ctypes.Structure):
        _fields_ = [("ntypes", ctypes.c_int32), ("rcut", ctypes.c_double), ("rcut_smth", ctypes.c_double),
                    ("sel", ctypes.c_void_p), ("emb_s1", ctypes.c_int32), ("m_axis", ctypes.c_int32),
                    ("fit_width", ctypes.c_int32), ("emb", ctypes.c_void_p), ("fit", ctypes.c_void_p)]
    d = Desc(1, 6.0, 0.5, None, 25, 16, 240, None, None)
    assert lib.dpb_model_create(ctypes.byref(d), 7, ctypes.byref(out)) == -1      # not a dpb_precision
    assert lib.dpb_model_create(ctypes.byref(d), 2, ctypes.byref(out)) == -1      # BF16 is built: null sel / weights
    assert lib.dpb_model_create(ctypes.byref(d), 1, ctypes.byref(out)) == -1      # TF32 is built: null sel / weights
    assert lib.dpb_model_create(ctypes.byref(d), 0, ctypes.byref(out)) == -1      # null sel / weights
    assert not out.value


def test_sass_is_sm100a_with_fp64_tensor_core_tiles():
    """The shipped library holds sm_100a code only, and the fused kernels use the fp64 tensor-core path (DMMA)."""
    import shutil
    import subprocess
    from paper_2004_11658_b200 import build
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    out = subprocess.run([cuobjdump, "-lelf", build.build()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_mixed_precision_kernels_use_tcgen05_and_tmem():
    """The DPB_TF32 kernels are Blackwell-native: tcgen05.mma (SASS UTC*MMA), TMEM loads (LDTM) and bulk copies
    (UBLKCP) appear in the SASS of the embedding / fitting objects; no legacy HMMA path."""
    import shutil
    import subprocess
    from paper_2004_11658_b200 import build
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    build.build()
    for obj, must in (("embed_tc.o", ("UTCHMMA", "LDTM")), ("fit_tc.o", ("UTCHMMA", "LDTM", "UBLKCP"))):
        sass = subprocess.run([cuobjdump, "-sass", os.path.join(build.OBJ, obj)], capture_output=True, text=True).stdout
        for mnem in must:
            assert mnem in sass, (obj, mnem)
        assert " HMMA" not in sass


def test_binding_fails_loudly_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import numpy as np
    from paper_2004_11658_b200 import DPModel, DPBError
    with pytest.raises(DPBError):
        DPModel(1, 6.0, 0.5, [8], 4, 2, 8, np.zeros(100), np.zeros(1000))


def test_product_never_imports_the_oracle():
    """The product path must not route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2004_11658_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "libdpo" not in text, f
                assert "dpo.h" not in text, f

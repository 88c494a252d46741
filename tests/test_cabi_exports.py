"""The C-ABI library builds for sm_100a, loads without a GPU, exports every symbol that
include/amrhydro.h declares, and refuses to run without a device (no CPU fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_0910_5547_b200 import build, binding
    build.build()
    return binding.load_library()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "amrhydro.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(amrhydro_[a-z_]+)\s*\(", text)))


def test_header_and_binding_agree(lib):
    from paper_0910_5547_b200 import binding
    names = declared_symbols()
    assert len(names) >= 20
    assert sorted(binding.EXPORTS) == names
    for n in names:
        assert hasattr(lib, n), n


def test_descriptor_struct_is_128_bytes():
    from paper_0910_5547_b200 import binding
    assert ctypes.sizeof(binding.PatchDesc) == 128


def test_no_cpu_fallback_without_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    lib.amrhydro_create.restype = ctypes.c_void_p
    assert not lib.amrhydro_create(1.4, 5, 16, 2)          # NULL: no device, nothing to fall back to
    from paper_0910_5547_b200 import binding, workloads as wl
    with pytest.raises(binding.AmrHydroError):
        binding.AmrHydro(wl.uniform_hierarchy(1), 1.4, 5)


def test_create_rejects_bad_arguments(lib):
    lib.amrhydro_create.restype = ctypes.c_void_p
    for args in ((1.0, 5, 16, 2), (1.4, 6, 16, 2), (1.4, 5, 32, 2), (1.4, 5, 16, 3)):
        assert not lib.amrhydro_create(*args)


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_0910_5547_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "liboracle" not in src, f
    src = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "amr_oracle.cpp")).read()
    assert "import paper_0910_5547_b200" not in src and "from paper_0910_5547_b200" not in src and "amrhydro.h" not in src

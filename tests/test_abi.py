"""CPU-side checks of the C-ABI boundary: the library builds/loads without a GPU, exports every
symbol include/sdm.h declares, and its host logic (sizing, argument checks) behaves."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2101_06318_b200 import build, binding
    build_path = build.build()
    assert os.path.exists(build_path)
    return binding.load_library()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "sdm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sdm_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    from paper_2101_06318_b200 import binding
    declared = _declared_symbols()
    assert declared == sorted(binding.SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name


def test_no_torch_types_and_extern_c_in_header():
    text = open(os.path.join(ROOT, "include", "sdm.h")).read()
    assert 'extern "C"' in text and "torch" not in text and "at::" not in text


def test_version_and_workspace_sizing(lib):
    assert lib.sdm_version() == 2000
    assert lib.sdm_workspace_bytes(0, 1) == 0
    assert lib.sdm_workspace_bytes(10, 0) == 0
    assert lib.sdm_workspace_bytes(2 ** 31, 1) == 0
    small = lib.sdm_workspace_bytes(1000, 4)
    big = lib.sdm_workspace_bytes(2 ** 26, 512 * 512)
    assert 0 < small < big
    # state (20 B) + idx (4 B) + order (4 B) per droplet dominate; everything else is < 10 %
    assert 28 * 2 ** 26 <= big < 1.1 * 28 * 2 ** 26
    assert small % 256 == 0 and big % 256 == 0
    # extensive attributes: 8 B per droplet and extra row; n_attr = 1 is the plain layout
    assert lib.sdm_workspace_bytes_attr(1000, 4, 1) == small
    assert lib.sdm_workspace_bytes_attr(1000, 4, 0) == 0 and lib.sdm_workspace_bytes_attr(1000, 4, 9) == 0
    a3 = lib.sdm_workspace_bytes_attr(2 ** 20, 4, 3) - lib.sdm_workspace_bytes_attr(2 ** 20, 4, 1)
    assert 2 * 8 * 2 ** 20 <= a3 < 2 * 8 * 2 ** 20 + 4096


def test_create_rejects_bad_arguments_without_touching_the_gpu(lib):
    h = C.c_void_p()
    assert lib.sdm_create(None, 10, 1, None, 0, None) == -1
    assert lib.sdm_create(C.byref(h), 0, 1, None, 0, None) == -1
    assert lib.sdm_create(C.byref(h), 10, 1, None, 1 << 20, None) == -1            # NULL workspace
    assert lib.sdm_create(C.byref(h), 10, 1, C.c_void_p(128), 1 << 30, None) == -1  # misaligned
    assert lib.sdm_create(C.byref(h), 10, 1, C.c_void_p(256), 16, None) == -1       # too small
    assert b"workspace" in lib.sdm_last_error(None)
    assert h.value is None
    assert lib.sdm_create_attr(C.byref(h), 10, 1, 9, C.c_void_p(256), 1 << 30, None) == -1   # n_attr > SDM_MAX_ATTR
    assert lib.sdm_destroy(None) == -1 and lib.sdm_set_option(None, 1, 1) == -1


def test_binding_fails_loudly_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2101_06318_b200 import SDM
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        SDM(16, 1)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2101_06318_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no oracle", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2101_06318_b200 import" not in src and "import paper_2101_06318_b200" not in src
            assert "libsdm" not in src and "include/sdm.h" not in src

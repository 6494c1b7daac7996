"""CPU-side checks of the boundary: libpn.so builds, loads, exports every symbol include/pn.h declares,
and its host-only logic (shape checks, error texts, workspace sizing) behaves.  No compute calls."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1908_03301_b200 import build, pn
    build.build()
    return pn.load_library()


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "pn.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b(pn_[a-z_0-9]+)\s*\(", src)
    return sorted(set(names))


def test_header_symbols_exported(lib):
    from paper_1908_03301_b200 import pn
    declared = _declared_functions()
    assert len(declared) >= 10
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/pn.h but not exported by libpn.so"
    assert sorted(pn.SYMBOLS) == declared


def test_header_cites_the_paper():
    src = open(os.path.join(ROOT, "include", "pn.h")).read()
    for needle in ("P:53", "P:57", "P:85", "eq.(4)", "forward-bond", "PN_ERR_VALUE"):
        assert needle.lower() in src.lower()


def test_workspace_bytes(lib):
    assert lib.pn_workspace_bytes(0, 4, 4) == 0
    assert lib.pn_workspace_bytes(4, -1, 4) == 0
    assert lib.pn_workspace_bytes(2048, 2048, 2048) == 0          # more than 2^31 padded nodes
    small = lib.pn_workspace_bytes(64, 64, 1)
    big = lib.pn_workspace_bytes(512, 512, 512)
    assert 0 < small < 1 << 20
    n = 512 ** 3
    assert 70 * n < big < 80 * n                                   # ~77 B per node
    assert big < 20 * (1 << 30)                                    # fits a 180 GB B200 many times over
    # padded pitch: 17 -> 20 columns
    assert lib.pn_workspace_bytes(17, 9, 5) > lib.pn_workspace_bytes(16, 9, 5)


def test_strerror(lib):
    from paper_1908_03301_b200 import pn
    texts = {c: pn.strerror(c) for c in range(-7, 3)}
    assert len(set(texts.values())) == len(texts)
    assert pn.strerror(12345) == "unknown code"


def test_create_argument_errors(lib):
    from paper_1908_03301_b200 import pn
    h = ctypes.c_void_p()
    assert lib.pn_create(None, 8, 8, 8, 0, None, ctypes.c_void_p(256), 1 << 30) == pn.PN_ERR_ARG
    assert lib.pn_create(ctypes.byref(h), 0, 8, 8, 0, None, ctypes.c_void_p(256), 1 << 30) == pn.PN_ERR_ARG
    assert lib.pn_create(ctypes.byref(h), 8, 8, 8, 0, None, None, 1 << 30) == pn.PN_ERR_WORKSPACE
    assert lib.pn_create(ctypes.byref(h), 8, 8, 8, 0, None, ctypes.c_void_p(264), 1 << 30) == pn.PN_ERR_WORKSPACE
    assert lib.pn_create(ctypes.byref(h), 8, 8, 8, 0, None, ctypes.c_void_p(256), 16) == pn.PN_ERR_WORKSPACE
    assert not h.value


def test_null_handles(lib):
    from paper_1908_03301_b200 import pn
    assert lib.pn_destroy(None) == pn.PN_OK
    assert lib.pn_solve(None, 0, 1e-10, None) == pn.PN_ERR_ARG
    assert lib.pn_set_option(None, 0, 1.0) == pn.PN_ERR_ARG
    assert lib.pn_flux(None, None, None, None, None) == pn.PN_ERR_ARG
    assert lib.pn_launch_count(None) == 0


def test_no_cuda_device_fails_loudly(lib):
    """Without a GPU the product path must raise, never fall back to a CPU path."""
    import torch
    from paper_1908_03301_b200 import pn
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(RuntimeError):
        pn.Network(8, 8, 8)
    h = ctypes.c_void_p()
    rc = lib.pn_create(ctypes.byref(h), 8, 8, 8, 0, None, ctypes.c_void_p(256), 1 << 30)
    assert rc == pn.PN_ERR_CUDA


def test_product_does_not_import_oracle():
    """The oracle is test infrastructure: nothing under the package may import or read it."""
    pkg = os.path.join(ROOT, "paper_1908_03301_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "pn_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1908_03301_b200" not in text.replace("(`paper_1908_03301_b200/`)", ""), f


def test_noalloc_argument_errors(lib):
    """pn_dissipation_noalloc refuses bad shapes and sizes beyond its fixed scratch array before any CUDA call."""
    from paper_1908_03301_b200 import pn
    p = ctypes.c_void_p(256)
    f = lib.pn_dissipation_noalloc
    assert f(0, 4, 4, p, p, p, p, 0, p, 0, None) == pn.PN_ERR_ARG
    assert f(4, 4, 4, None, p, p, p, 0, p, 0, None) == pn.PN_ERR_ARG
    assert f(4, 4, 4, p, p, p, p, 0, None, 0, None) == pn.PN_ERR_ARG
    assert f(4, 4, 4, p, p, None, p, 0, p, 0, None) == pn.PN_ERR_ARG          # 3D without gz
    assert f(4, 4, 1, p, p, p, p, 0, p, 0, None) == pn.PN_ERR_ARG             # 2D with gz
    assert f(4, 4, 4, p, p, p, p, 8, p, 0, None) == pn.PN_ERR_ARG             # mask has three bits
    assert f(4, 4, 4, p, p, p, p, 0, p, -1, None) == pn.PN_ERR_ARG
    assert f(1024, 1024, 257, p, p, p, p, 0, p, 0, None) == pn.PN_ERR_TOO_LARGE
    assert f(1 << 20, 1 << 20, 1, p, p, None, p, 0, p, 0, None) == pn.PN_ERR_TOO_LARGE
    assert f(2147483647, 2147483647, 2147483647, p, p, p, p, 0, p, 0, None) == pn.PN_ERR_TOO_LARGE
    assert pn.PN_NOALLOC_MAX_NODES == 1024 * 1024 * 256
    assert "PN_NOALLOC_MAX_NODES" in pn.strerror(pn.PN_ERR_TOO_LARGE)

"""CPU-side checks of the boundary: libnif.so builds, loads and exports every symbol that
include/nif.h declares; host-only entry points work; kernels refuse to run without an sm_100
GPU instead of falling back (no compute calls here)."""
import ctypes as C
import re
from pathlib import Path

import pytest
import torch

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    from paper_2604_24666_b200 import build
    build.build()
    import paper_2604_24666_b200 as nif
    return nif.lib()


def _declared():
    text = (ROOT / "include" / "nif.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(nif_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared()
    assert {"nif_build_deformed_bvh", "nif_query", "nif_net_create", "nif_query_host"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/nif.h but not exported by libnif.so"


def test_header_is_plain_c(tmp_path):
    import subprocess
    src = tmp_path / "t.c"
    src.write_text('#include "nif.h"\nint main(void){ nif_query_out o; (void)o; return NIF_N_OUT == 12 ? 0 : 1; }\n')
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", str(ROOT / "include"), "-c", str(src),
                           "-o", str(tmp_path / "t.o")])


def test_host_only_entry_points(lib):
    import paper_2604_24666_b200 as nif
    small = nif.nif_bvh_workspace_bytes(16, 1088)
    big = nif.nif_bvh_workspace_bytes(16, 16 ** 3)
    assert 0 < small <= big and small % 256 == 0
    assert nif.nif_bvh_workspace_bytes(256, 860_000) < 2 << 30
    n = C.c_size_t()
    assert lib.nif_bvh_workspace_bytes(1, 10, C.byref(n)) == -1          # nv out of range
    assert lib.nif_bvh_workspace_bytes(1024, 10, C.byref(n)) == -1
    assert lib.nif_bvh_workspace_bytes(16, 10, None) == -1
    assert nif.nif_query_workspace_bytes(0) >= 64
    assert nif.nif_query_workspace_bytes(1 << 20) >= 64 + 4 * (1 << 20)
    assert lib.nif_query_workspace_bytes(-1, C.byref(n)) == -1
    assert nif.nif_query_multi_workspace_bytes(1 << 20) >= nif.nif_query_workspace_bytes(1 << 20) + 8 * (1 << 20)
    assert lib.nif_query_multi_workspace_bytes(-1, C.byref(n)) == -1
    assert lib.nif_error_string(0) == b"ok"
    for s in range(-5, 0):
        assert lib.nif_error_string(s) not in (b"ok", b"unknown status")
    assert lib.nif_error_string(-99) == b"unknown status"
    assert nif.nif_kernel_launch_count() >= 0


def test_argument_validation_without_touching_the_device(lib):
    assert lib.nif_build_deformed_bvh(None, None, None, 0, None, None) == -1
    assert lib.nif_net_create(None, None, None, None, None) == -1
    assert lib.nif_query(None, None, None, None, None, 0, 0, None) == -1
    assert lib.nif_query_host(None, None, None, None, None, 0) == -1
    assert lib.nif_query_multi(None, None, None, None, None, 4, None, 0, 0, None) == -1
    h = C.c_void_p()
    assert lib.nif_stage_create(0, C.byref(h)) == -1


def test_static_query_checks_its_limit_before_any_device_work(lib):
    # nif_query_static: argument errors and the size limit are decided on the host, before the first CUDA call
    from paper_2604_24666_b200 import binding as B
    assert lib.nif_query_static(None, None, None, None, 0, None) == -1
    fake = C.c_void_p(256)                                   # handles are only null-checked before the limit check
    q = B._QueryOut()
    for name, _ in B._QueryOut._fields_:
        setattr(q, name, 256)
    for n, expect in ((B.NIF_STATIC_MAX_RAYS + 1, -7), (-1, -1), (0, 0)):
        rb = B._RayBatch(n, 256, 256)
        assert lib.nif_query_static(fake, fake, C.byref(rb), C.byref(q), 0, None) == expect, n
    assert b"NIF_STATIC_MAX_RAYS" in lib.nif_error_string(-7)


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_gpu_means_unsupported_not_a_fallback(lib):
    import numpy as np
    from paper_2604_24666_b200 import binding as B
    occ = np.ones(8, np.uint8)
    vs = B._VoxelSet(2, occ.ctypes.data)
    dp = B._DeformParams(0.0, 0.0)
    ws = np.zeros(1 << 16, np.uint8)
    base = ws.ctypes.data + (-ws.ctypes.data) % 256
    h = C.c_void_p()
    rc = lib.nif_build_deformed_bvh(C.byref(vs), C.byref(dp), base, 1 << 15, None, C.byref(h))
    assert rc == -2 and not h.value                                   # NIF_ERR_UNSUPPORTED
    assert lib.nif_stage_create(16, C.byref(h)) == -2


def test_binding_fails_loudly_when_library_is_missing(monkeypatch, tmp_path):
    from paper_2604_24666_b200 import binding as B
    monkeypatch.setattr(B, "_lib", None)
    monkeypatch.setattr(B, "LIB_PATH", tmp_path / "nope.so")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        B.lib()

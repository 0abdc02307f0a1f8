"""CPU-only checks of the C-ABI boundary: the library builds/loads without a GPU, exports
every symbol include/affinescan.h declares, and rejects bad arguments with status codes
before touching the device (no compute calls here)."""
import ctypes
import os

import paper_2606_00601_b200 as lib
from paper_2606_00601_b200 import build as libbuild

EXPECTED = {
    "affine_scan", "affine_scan_ex", "affine_scan_host",
    "selective_scan_fwd", "selective_scan_fwd_ex", "selective_scan_fwd_host",
    "selective_scan_fwd_ext", "selective_scan_fwd_ext_host", "selective_scan_fwd_gated",
    "affinescan_reset_mask_from_cu_seqlens", "selective_scan_bwd",
    "selective_scan_slice_aggregate", "affinescan_compose_carry",
    "affinescan_status_string", "affinescan_last_cuda_error", "affinescan_last_variant",
    "affinescan_launch_count", "affinescan_version", "affinescan_release_cache",
    "affinescan_set_option",
    "affine_scan_static_scratch", "affine_scan_static_scratch_max_elements",
    "affinescan_cached_scratch_buffers",
    "selective_scan_bwd_ws", "selective_scan_bwd_workspace_bytes",
}


def test_library_builds_and_loads():
    path = libbuild.build()
    assert os.path.exists(path)
    assert lib.load() is not None
    assert lib.version() >= 200


def test_exports_every_declared_symbol():
    declared = set(lib.declared_symbols())
    assert declared == EXPECTED, declared ^ EXPECTED
    raw = ctypes.CDLL(lib.library_path())
    for name in declared:
        assert getattr(raw, name) is not None, name


def test_header_cites_the_paper_for_each_operation():
    with open(os.path.join(libbuild.ROOT, "include", "affinescan.h")) as f:
        text = f.read()
    for needle in ("P:86", "P:90", "P:69", "P:81", "P:73", "BJ", "caller owns"):
        assert needle in text, needle


def test_status_strings():
    assert lib.status_string(0) == "ok"
    seen = {lib.status_string(i) for i in range(7)}
    assert len(seen) == 7
    assert lib.status_string(99) == "unknown status"


def test_argument_validation_without_device_work():
    L = lib.load()
    n = ctypes.c_void_p(None)
    p = ctypes.c_void_p(0x1000)  # never dereferenced: validation fails first
    # dtype
    assert L.affine_scan(p, p, n, p, n, 4, 8, 7, n) == 3
    assert L.selective_scan_fwd(p, p, p, p, p, n, n, p, n, 1, 1, 16, 8, -1, n) == 3
    # shape
    assert L.affine_scan(p, p, n, p, n, -1, 8, 0, n) == 2
    assert L.affine_scan(p, p, n, p, n, 4, -8, 0, n) == 2
    assert L.affine_scan(p, p, n, p, n, 1 << 40, 1 << 40, 0, n) == 2   # product overflows
    assert L.selective_scan_fwd(p, p, p, p, p, n, n, p, n, -1, 1, 16, 8, 0, n) == 2
    # N outside [1, 64]
    assert L.selective_scan_fwd(p, p, p, p, p, n, n, p, n, 1, 1, 0, 8, 0, n) == 4
    assert L.selective_scan_fwd(p, p, p, p, p, n, n, p, n, 1, 1, 65, 8, 0, n) == 4
    # NULL required pointers
    assert L.affine_scan(n, p, n, p, n, 4, 8, 0, n) == 1
    assert L.affine_scan(p, p, n, n, n, 4, 8, 0, n) == 1
    assert L.selective_scan_fwd(p, p, n, p, p, n, n, p, n, 1, 1, 16, 8, 0, n) == 1
    assert L.selective_scan_fwd_host(p, p, p, p, p, n, n, n, n, 1, 1, 16, 8, 0, n) == 1
    # empty problems are OK and need no device
    assert L.affine_scan(n, n, n, n, n, 0, 8, 0, n) == 0
    assert L.selective_scan_fwd(n, n, n, n, n, n, n, n, n, 0, 64, 16, 8, 0, n) == 0
    assert L.affinescan_last_variant() == 0


def test_binding_has_no_fallback_and_never_imports_the_oracle():
    pkg = os.path.dirname(lib.__file__)
    for name in os.listdir(pkg):
        if name.endswith(".py"):
            with open(os.path.join(pkg, name)) as f:
                src = f.read()
            assert "import oracle" not in src and "from oracle" not in src, name
    for root, _, files in os.walk(os.path.join(pkg, "csrc")):
        for name in files:
            with open(os.path.join(root, name)) as f:
                assert "oracle" not in f.read().lower(), name
    # and the oracle never imports the CUDA package
    odir = os.path.join(libbuild.ROOT, "oracle")
    for name in os.listdir(odir):
        if name.endswith((".py", ".c")):
            with open(os.path.join(odir, name)) as f:
                src = f.read()
            assert "import paper_2606_00601_b200" not in src
            assert "from paper_2606_00601_b200" not in src

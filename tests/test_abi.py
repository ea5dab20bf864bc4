"""CPU-side checks of the C-ABI boundary (no compute without a GPU): libhva.so builds, loads, exports every symbol that
include/hva.h declares (and the Python binding lists the same set), the host-only entry points answer, and the argument
checks return the documented error codes before anything touches CUDA."""
import ctypes as C
import os
import re

import pytest

from paper_2607_03012_b200 import binding as b, build, inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "hva.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hva_[a-z_0-9]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    build.build(force=False)
    return b.lib()


def test_every_declared_symbol_is_exported_and_bound(lib):
    names = _declared()
    assert len(names) >= 20
    for n in names:
        assert getattr(lib, n) is not None, n
    assert sorted(b.EXPORTS) == names                      # the binding covers exactly the header


def test_host_only_entry_points(lib):
    assert lib.hva_version() >= 100
    assert lib.hva_strerror(0) == b"ok" and b"invalid" in lib.hva_strerror(-1)
    wl = inputs.C4
    shape, cfg = b.make_shape(wl), b.make_config(wl)
    assert b.hva_num_clusters(shape, wl.cell) == 990       # 11 x 9 x 10 (BASELINE.json configs[3])
    ws, st = b.hva_workspace_bytes(shape, cfg), lib.hva_state_bytes(C.byref(shape), C.byref(cfg))
    assert ws > 2 * wl.heads * wl.n * wl.D * 2 and 0 < st < ws          # K', V' live in the workspace (Q' is gathered inside the kernel)
    assert ws < 3 * wl.heads * wl.n * wl.D * 2
    L = b.hva_plan_describe(24, wl.n, 990, 990, 128)
    assert L.work_cap >= -(-wl.n // 128) + 990 and L.total > 3 * 24 * wl.n * 4
    assert lib.hva_cluster_workspace_bytes(C.byref(shape), (C.c_int32 * 3)(*wl.cell), (C.c_int32 * 3)(*wl.win)) > 0
    assert lib.hva_merge_workspace_bytes(24, 990, 990) > 24 * 990 * 31 * 4
    assert lib.hva_cluster_update_workspace_bytes(C.byref(shape), 990, 17820) > 24 * 17820 * 8


def test_argument_checks_return_error_codes_without_cuda(lib):
    wl = inputs.C2
    shape, cfg = b.make_shape(wl), b.make_config(wl)
    null = C.c_void_p(0)
    assert lib.hva_forward(C.byref(shape), C.byref(cfg), null, null, null, null, 0, null, null, null, C.c_size_t(0), null) == -1
    assert lib.hva_cluster(C.byref(shape), (C.c_int32 * 3)(1, 1, 1), (C.c_int32 * 3)(3, 3, 3), 0, null, null, null, null, null, null,
                           null, null, C.c_size_t(0), null) == -1
    assert lib.hva_build_mask(1, 8, 8, 48, null, null, null, C.c_float(1.0), C.c_float(0.9), C.c_float(0.0), null, null, C.c_size_t(0), null) == -1
    bad = b.make_shape(wl)
    bad.D = 96
    assert lib.hva_workspace_bytes(C.byref(bad), C.byref(cfg)) == 0
    assert lib.hva_merge_workspace_bytes(0, 8, 8) == 0


def test_state_and_plan_layout_queries(lib):
    """hva_state_describe / hva_plan_workspace_bytes: the binding no longer mirrors private layouts of api.cu / plan.cu."""
    wl = inputs.C4
    shape, cfg = b.make_shape(wl), b.make_config(wl, subset_frac=0.15)
    L = b.hva_state_layout()
    assert lib.hva_state_describe(C.byref(shape), C.byref(cfg), C.byref(L)) == 0
    assert L.total == lib.hva_state_bytes(C.byref(shape), C.byref(cfg))
    assert list(L.n_clusters) == [990, 990] and L.m == 17820            # floor(0.15 * 118800 + 1/2)  (R-H2)
    offs = sorted([L.assign[0], L.mu[0], L.sums[0], L.sizes[0], L.subset[0], L.assign[1], L.mu[1], L.sums[1], L.sizes[1], L.subset[1]])
    assert offs[0] == 0 and all(o % 256 == 0 for o in offs) and len(set(offs)) == 10 and offs[-1] < L.total
    assert L.mu[0] - L.assign[0] >= 24 * wl.n * 4 and L.sums[0] - L.mu[0] >= 24 * 990 * 128 * 4
    assert lib.hva_state_describe(C.byref(shape), C.byref(cfg), C.c_void_p(0)) == -1
    assert lib.hva_plan_workspace_bytes(24, wl.n, 990, 990) >= 24 * 117 * 990 * 4
    assert lib.hva_plan_workspace_bytes(0, wl.n, 990, 990) == 0


def test_host_call_validates_before_enqueueing(lib):
    """hva_forward_host: bad arguments / a short workspace are reported before any copy is enqueued (no CUDA needed)."""
    wl = inputs.C2
    shape, cfg = b.make_shape(wl), b.make_config(wl)
    null, one = C.c_void_p(0), C.c_void_p(16)
    assert lib.hva_forward_host(C.byref(shape), C.byref(cfg), null, one, one, one, 0, null, one, one, C.c_size_t(1 << 40), null) == -1
    assert lib.hva_forward_host(C.byref(shape), C.byref(cfg), one, one, one, one, 7, null, one, one, C.c_size_t(1 << 40), null) == -1
    assert lib.hva_forward_host(C.byref(shape), C.byref(cfg), one, one, one, one, 1, null, one, one, C.c_size_t(1 << 40), null) == -1  # intermediate without state
    assert lib.hva_forward_host(C.byref(shape), C.byref(cfg), one, one, one, one, 0, null, one, one, C.c_size_t(1024), null) == -2


def test_library_reads_no_environment_and_keeps_no_probe_pointers():
    """SURVEY section 5 'no env vars, no global state': kernel selection is an explicit `flags` argument."""
    csrc = os.path.join(ROOT, "paper_2607_03012_b200", "csrc")
    for f in sorted(os.listdir(csrc)):
        src = open(os.path.join(csrc, f)).read()
        assert "getenv" not in src and "strtoull" not in src, f
    cfg = b.make_config(inputs.C2, flags=b.HVA_FLAG_ATTN_SIMT | b.HVA_FLAG_MERGE_SIMT)
    assert cfg.flags == 10 and C.sizeof(b.hva_config) == 4 * (12 + 12) and b.HVA_FLAG_Q_UNPERMUTED == 16


def test_static_scratch_plan_limit_is_checked_before_anything_else(lib):
    """hva_build_plan_static: sizes beyond the built-in array are refused with HVA_ELIMIT before any CUDA call (so also here,
    without a GPU); the limit is the header's constant."""
    import re
    hdr = open(os.path.join(ROOT, "include", "hva.h")).read()
    m = re.search(r"#define HVA_PLAN_STATIC_SCRATCH_BYTES \((\d+)u << (\d+)\)", hdr)
    assert m and lib.hva_build_plan_static_limit() == int(m.group(1)) << int(m.group(2)) == 32 << 20
    assert lib.hva_plan_workspace_bytes(24, 118800, 990, 990) <= lib.hva_build_plan_static_limit()      # C4 fits
    assert lib.hva_plan_workspace_bytes(64, 118800, 990, 990) > lib.hva_build_plan_static_limit()
    z = C.c_void_p(0)
    rc = lib.hva_build_plan_static(64, 118800, 990, 990, z, z, z, z, z, z, z, 128, 128, z, C.c_size_t(0), z)
    assert rc == -5 and b"static" in lib.hva_strerror(rc)
    assert lib.hva_build_plan_static(0, 118800, 990, 990, z, z, z, z, z, z, z, 128, 128, z, C.c_size_t(0), z) == -1
    # the path allocates nothing: no cudaMalloc / cudaFree in the translation unit that holds it
    src = open(os.path.join(ROOT, "paper_2607_03012_b200", "csrc", "plan.cu")).read()
    assert "cudaMalloc" not in src.replace("cudaMalloc /", "") and "cudaFree(" not in src
    assert "cudaGetSymbolAddress(&p, g_plan_static_scratch)" in src

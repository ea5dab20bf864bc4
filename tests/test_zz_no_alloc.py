"""hva_build_plan_static (include/hva.h): the plan stage with the library's built-in device scratch array instead of a
caller-provided workspace, for callers that may not allocate.  Its output must equal hva_build_plan's bit for bit (the plan is
integer / index work: the tolerance of every plan test here is exact equality), on two calls in a row that use the shared
array with DIFFERENT layouts (so whatever the first call left behind lies under the second call's histograms), and the
call itself must not change the amount of free device memory.

Collected last on purpose (file name): the suite runs with pytest -x.  Passes alone in a fresh process and after the others:
it keeps no state besides the library's own array, which no other entry point touches.
"""
import dataclasses
import math

import pytest
import torch

from paper_2607_03012_b200 import inputs

pytestmark = pytest.mark.gpu


def _b():
    from paper_2607_03012_b200 import binding
    if not torch.cuda.is_available():
        pytest.fail("the gpu tests need a CUDA device")
    return binding


def _stage_inputs(b, wl, heads, merge_rounds):
    """Seeded synthetic Q, K of `heads` through the GPU stages up to merging: what hva_build_plan consumes."""
    Q, K, _ = inputs.make_qkv(wl, heads=heads)
    shape = b.make_shape(wl, heads=len(heads))
    cq = b.hva_cluster(shape, wl.cell, wl.win, wl.iters, Q.cuda().contiguous(), want_sums=False, want_lowe=False)
    ck = b.hva_cluster(shape, wl.cell, wl.win, wl.iters, K.cuda().contiguous(), want_sums=False, want_lowe=False)
    mask = b.hva_build_mask(cq["mu"], ck["mu"], ck["sizes"], 1.0 / math.sqrt(wl.D), wl.top_p)
    gof, ng, gm = b.hva_merge(cq["sizes"], ck["sizes"], mask, wl.tile[0], wl.tile[1], merge_rounds, seed=wl.seed)
    return dict(n=wl.n, assign_q=cq["assign"], assign_k=ck["assign"], sizes_q=cq["sizes"], sizes_k=ck["sizes"], group_of=gof,
                n_groups=ng, gmask=gm, tile_q=wl.tile[0], tile_k=wl.tile[1])


def _same_plan(pa, pb):
    assert pa.L.total == pb.L.total
    assert torch.equal(pa.buf, pb.buf), "plan buffers differ"
    # and the named arrays, so that a failure says which one
    for k in ("perm_q", "inv_perm_q", "perm_k", "koff", "goff", "gid"):
        assert torch.equal(getattr(pa, k), getattr(pb, k)), k
    assert pa.stats_dicts() == pb.stats_dicts()


def test_static_scratch_plan_equals_workspace_plan_on_two_calls_in_a_row():
    b = _b()
    # call 1: C2 (8 heads x 6912 tokens, 144 clusters, 128-row tiles, several sort tiles and a ragged one), merging on
    # call 2: another lattice / head count / tile size / cluster count and merging off -> the array is laid out differently
    wl1 = inputs.CONFIGS["C2"]
    wl2 = dataclasses.replace(inputs.CONFIGS["C2"], T=7, H=22, W=30, cell=(2, 4, 5), tile=(64, 64), seed=11)   # non-dividing lattice
    a1 = _stage_inputs(b, wl1, list(range(8)), merge_rounds=3)
    a2 = _stage_inputs(b, wl2, [0, 3, 5], merge_rounds=0)
    ref1 = b.hva_build_plan(**a1)
    ref2 = b.hva_build_plan(**a2)
    out1 = torch.zeros(ref1.L.total, dtype=torch.uint8, device="cuda")
    out2 = torch.zeros(ref2.L.total, dtype=torch.uint8, device="cuda")
    out3 = torch.zeros(ref2.L.total, dtype=torch.uint8, device="cuda")
    torch.cuda.synchronize()
    got1 = b.hva_build_plan_static(**a1, out=out1)
    got2 = b.hva_build_plan_static(**a2, out=out2)          # right behind call 1 on the same stream, no sync in between
    torch.cuda.synchronize()
    _same_plan(got1, ref1)
    _same_plan(got2, ref2)
    assert int(a1["n_groups"].sum()) > 0 and int(a2["n_groups"].sum()) > 0
    # a third call (everything it launches has run before): the driver's free-memory figure must not move across it
    free_before, _ = torch.cuda.mem_get_info()
    got3 = b.hva_build_plan_static(**a2, out=out3)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    _same_plan(got3, ref2)
    assert free_after == free_before, (free_before, free_after)


def test_static_scratch_plan_rejects_sizes_beyond_its_array():
    b = _b()
    lim = b.lib().hva_build_plan_static_limit()
    assert lim == 32 << 20
    # 64 heads of the C4 lattice need 59 MB of sort histograms: rejected up front (nothing is dereferenced or enqueued)
    need = b.lib().hva_plan_workspace_bytes(64, 118800, 990, 990)
    assert need > lim
    import ctypes as C
    z = C.c_void_p(0)
    rc = b.lib().hva_build_plan_static(64, 118800, 990, 990, z, z, z, z, z, z, z, 128, 128, z, C.c_size_t(0), z)
    assert rc == -5 and b"static" in b.lib().hva_strerror(rc)
    torch.cuda.synchronize()

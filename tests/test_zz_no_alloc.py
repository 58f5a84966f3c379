"""scw_eval_points_noalloc: the plane-wave point sum for callers that cannot allocate GPU memory.

Some users of libscw run where device memory can no longer be had: a plug-in inside an application whose memory pool
already owns the whole GPU, a real-time loop that must not enter the allocator (cudaMalloc locks the process and may
stall the device), an out-of-memory handler.  They cannot give scw_eval_points the workspace it tabulates the plane
waves in.  scw_eval_points_noalloc keeps that table in a fixed array inside libscw.so (at most
SCW_POINTS_NOALLOC_MAX_J = 8192 waves) and allocates nothing; the caller still passes the inputs and the output.

What is checked here: the new entry point returns the field of the existing scw_eval_points (whose parity with the fp64
oracle is tests/test_gpu_parity.py's business) within the complex64 tolerance of this repository, 2e-4 relative
max-norm -- on TWO calls in a row with different tables and points, because the built-in array is shared and keeps the
previous call's contents; a second call that trusted them would be caught.  Also: no workspace is needed or touched,
the CUDA allocator is not entered during the calls, and a table above the limit is refused cleanly.

The file name sorts last on purpose: `pytest -x` stops at the first failure, so a failure here hides no other test.
It passes alone in a fresh process (the first call then does the per-device address look-up) and after the other tests.
"""
import ctypes

import numpy as np
import pytest
import torch

import scw_inputs as si

pytestmark = pytest.mark.gpu

TOL_C64 = 2e-4          # relative max-norm, the complex64 bar of every GPU parity test (BASELINE.json north_star)


@pytest.fixture(scope="module")
def scw():
    import paper_2404_07293_b200 as m
    m.lib()                                    # fail loudly if the extension is missing
    return m


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rel_err(got, ref):
    got = got.cpu().numpy().astype(np.complex128)
    ref = ref.cpu().numpy().astype(np.complex128)
    return float(np.abs(got - ref).max() / np.abs(ref).max())


def subset(pw, J):
    """The first J waves of a plane-wave table (scalars are kept)."""
    return {k: (v[:J] if isinstance(v, np.ndarray) else v) for k, v in pw.items()}


def test_noalloc_matches_eval_points_on_two_calls_in_a_row(scw):
    cfg = si.CONFIGS[3]                                        # 33 x 33 frequencies, 4356 plane waves
    pw_full = si.make_planewaves(cfg)
    # call 1: the whole table, a ragged point count, points shifted far from the origin (large per-axis maxima in the
    # table header); call 2: a shorter table and fewer points, so stale header maxima or stale table rows would show
    cases = [(pw_full, si.make_points(cfg, n=5000 + 37) + np.array([3.0e4, -2.0e4, 0.0])),
             (subset(pw_full, 1000), si.make_points(cfg, n=1500)[::-1].copy())]

    ref_ctx = scw.Context(0)                                   # existing path: table in a torch-allocated workspace
    refs = []
    for pw, xyz in cases:
        refs.append(scw.scw_eval_points(ref_ctx, scw.PlaneWaves.from_numpy(pw, "cuda"), dev(xyz)))
    torch.cuda.synchronize()

    ctx = scw.Context(0)                                       # a ctx that never gets a workspace
    tabs = [scw.PlaneWaves.from_numpy(pw, "cuda") for pw, _ in cases]
    pts = [dev(xyz) for _, xyz in cases]
    outs = [torch.full((p.shape[0], 3), float("nan"), dtype=torch.complex64, device="cuda") for p in pts]
    # start-up: the first call on a device looks up where the GPU keeps the built-in array (documented as set-up work)
    scw.scw_eval_points_noalloc(ctx, tabs[1], pts[1][:8], outs[1][:8])
    outs[1].fill_(float("nan"))
    torch.cuda.synchronize()
    mem0 = torch.cuda.memory_allocated(), torch.cuda.memory_reserved()
    free0 = torch.cuda.mem_get_info()[0]
    n0 = ctx.launch_count()
    for tab, p, out in zip(tabs, pts, outs):                   # two calls in a row on one stream, no sync between them
        assert scw.scw_eval_points_noalloc(ctx, tab, p, out) is out
    torch.cuda.synchronize()
    assert ctx.launch_count() - n0 == 4                        # table + sum, twice: the library's own kernels ran
    assert ctx.workspace_bytes() == 0                          # no workspace was registered behind our back
    assert (torch.cuda.memory_allocated(), torch.cuda.memory_reserved()) == mem0
    assert torch.cuda.mem_get_info()[0] >= free0               # nothing was taken from the device either
    for out, ref in zip(outs, refs):
        assert torch.isfinite(torch.view_as_real(out)).all()
        assert rel_err(out, ref) <= TOL_C64
    # the same calls again in the opposite order (the array now holds call 2's short table)
    for i in (1, 0):
        outs[i].fill_(float("nan"))
        scw.scw_eval_points_noalloc(ctx, tabs[i], pts[i], outs[i])
    torch.cuda.synchronize()
    for out, ref in zip(outs, refs):
        assert rel_err(out, ref) <= TOL_C64
    ctx.close()
    ref_ctx.close()


def test_noalloc_rejects_what_it_cannot_hold(scw):
    cfg = si.CONFIGS[3]
    pw = si.make_planewaves(cfg)
    reps = scw.SCW_POINTS_NOALLOC_MAX_J // pw["J"] + 1
    big = {k: (np.concatenate([v] * reps) if isinstance(v, np.ndarray) else v) for k, v in pw.items()}
    assert big["p"].shape[0] > scw.SCW_POINTS_NOALLOC_MAX_J
    ctx = scw.Context(0)
    xyz = dev(si.make_points(cfg, n=64))
    out = torch.zeros((64, 3), dtype=torch.complex64, device="cuda")
    with pytest.raises(scw.ScwError) as ei:                    # above the limit: refused, nothing enqueued or written
        scw.scw_eval_points_noalloc(ctx, scw.PlaneWaves.from_numpy(big, "cuda"), xyz, out)
    assert ei.value.status == 2 and "SCW_POINTS_NOALLOC_MAX_J" in str(ei.value)
    torch.cuda.synchronize()
    assert float(torch.view_as_real(out).abs().max()) == 0.0
    # exactly at the limit it is taken, and agrees with the workspace path
    edge = {k: (v[:scw.SCW_POINTS_NOALLOC_MAX_J] if isinstance(v, np.ndarray) else v) for k, v in big.items()}
    tab = scw.PlaneWaves.from_numpy(edge, "cuda")
    scw.scw_eval_points_noalloc(ctx, tab, xyz, out)
    ref = scw.scw_eval_points(ctx, tab, xyz)
    torch.cuda.synchronize()
    assert rel_err(out, ref) <= TOL_C64
    # the dense kind is not served
    lay = si.make_layer(si.CONFIGS[0])
    m = scw.binding.scw_modes()
    m.struct_size = ctypes.sizeof(scw.binding.scw_modes)
    m.kind = scw.binding.SCW_MODES_DENSE
    L = scw.Layer.from_numpy(lay, "cuda")
    m.layer = L.struct()
    assert ctx.L.scw_eval_points_noalloc(ctx._h, ctypes.byref(m), 64, scw.binding._p(xyz), scw.binding._p(out)) == 8
    ctx.close()

"""GPU edge cases and error paths of the C ABI: ragged shapes, padding, strides, empties, bad arguments."""
import ctypes

import numpy as np
import pytest
import torch

import oracle
import scw_inputs as si

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def scw():
    import paper_2404_07293_b200 as m
    m.lib()
    return m


@pytest.fixture(scope="module")
def ctx(scw):
    c = scw.Context(0)
    yield c
    c.close()


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rel_err(got, ref):
    return float(np.abs(np.asarray(got, dtype=np.complex128) - ref).max() / np.abs(ref).max())


def ragged_layer(U, Vn, J, dtype, seed, ldV_pad=0, with_c=True, with_dir=True):
    g = np.random.default_rng(seed)
    R = 3 * U * Vn
    V = np.full((J, R + ldV_pad), 9.0 + 9.0j, dtype=dtype)        # padding rows hold garbage on purpose
    V[:, :R] = ((g.standard_normal((J, R)) + 1j * g.standard_normal((J, R))) / np.sqrt(2 * U * Vn)).astype(dtype)
    dirs = np.where(g.uniform(0, 1, J) < 0.5, 1, -1).astype(np.int8)
    gamma = dirs * (g.uniform(0.0, 1.5, J) + 1j * g.uniform(0.0, 0.8, J))
    c = ((g.standard_normal(J) + 1j * g.standard_normal(J)) / np.sqrt(2)).astype(dtype) if with_c else None
    return dict(U=U, Vn=Vn, X=3.0, Y=4.5, lam=0.7, z_lo=-0.4, z_hi=0.9, V=V, gamma=gamma, c=c,
                dir=dirs if with_dir else None)


@pytest.fixture(scope="module")
def ctx_simt(scw):
    c = scw.Context(0)
    c.set_path(scw.SCW_PATH_SIMT)
    yield c
    c.close()


@pytest.mark.parametrize("path", ["auto", "simt"])
@pytest.mark.parametrize("dtype,tol", [(np.complex64, 2e-4), (np.complex128, 1e-10)])
@pytest.mark.parametrize("U,Vn,J,Nx,Ny,Fz", [(5, 3, 17, 37, 21, 3), (1, 1, 4, 5, 130, 1), (4, 6, 96, 129, 7, 35),
                                             (7, 2, 56, 300, 3, 18)])
def test_ragged_shapes_padding_and_defaults(scw, ctx, ctx_simt, path, dtype, tol, U, Vn, J, Nx, Ny, Fz):
    """Odd/even frequency counts, J not 4M, padded ldV/ldP, c = NULL, dir = NULL, non-uniform x/y,
    z outside the layer: every sample against Tier A.  path "auto": complex128 on the DMMA kernels, complex64 on
    tcgen05 where a tile fits; "simt": the CUDA-core kernels for both."""
    ctx = ctx if path == "auto" else ctx_simt
    lay = ragged_layer(U, Vn, J, dtype, seed=U * 100 + J, ldV_pad=3, with_c=(J % 2 == 0), with_dir=(J % 3 == 0))
    g = np.random.default_rng(5)
    x = np.sort(g.uniform(-4, 7, Nx))
    y = np.sort(g.uniform(-4, 7, Ny))
    z = np.linspace(-0.6, 1.1, Fz)                                  # includes z outside [z_lo, z_hi]
    ref = oracle.layer_grid(x=x, y=y, z=z, **lay)
    L = scw.Layer.from_numpy(lay, "cuda")
    R = 3 * U * Vn
    Pbuf = torch.full((Fz, R + 5), 7.0, dtype=L.V.dtype, device="cuda")
    scw.scw_assemble_spectra(ctx, L, dev(z), out=Pbuf)
    assert torch.all(Pbuf[:, R:] == 7.0)                            # padding of P untouched
    E = scw.scw_synthesize_grid(ctx, U=U, Vn=Vn, X=lay["X"], Y=lay["Y"], P=Pbuf, x=dev(x), y=dev(y))
    torch.cuda.synchronize()
    assert rel_err(E.cpu().numpy(), ref) <= tol
    E2 = scw.scw_sweep_wavelengths(ctx, [L], [dev(z)], dev(x), dev(y))[0]
    torch.cuda.synchronize()
    assert rel_err(E2.cpu().numpy(), ref) <= tol
    # dense point path on a ragged number of points
    xyz = oracle.grid_points(x, y, z)[:: max(1, (Nx * Ny * Fz) // 301)]
    Ep = scw.scw_eval_points(ctx, L, dev(xyz))
    torch.cuda.synchronize()
    refp = oracle.layer_samples(xyz=xyz, **lay)
    assert np.abs(Ep.cpu().numpy() - refp).max() / np.abs(ref).max() <= tol


@pytest.mark.parametrize("U,Vn,J,Fz,pad,n_inst", [(5, 3, 17, 3, 0, 1), (5, 3, 33, 9, 1, 2), (7, 9, 250, 20, 2, 3),
                                                   (9, 11, 131, 70, 3, 1), (3, 1, 2, 1, 0, 1),
                                                   (45, 50, 64, 4, 1, 1), (65, 41, 40, 3, 0, 2), (80, 80, 36, 2, 0, 1)])
def test_forced_tensor_path_ragged(scw, U, Vn, J, Fz, pad, n_inst):
    """SCW_PATH_TENSOR on shapes that are not multiples of any tile: odd and even ldV (the two TMA column maps),
    rows not a multiple of 128, J not a multiple of 32 (zero-filled boxes), Fz not a multiple of 8 and above one
    n tile, grouped instances, more than 40 frequencies per axis (two frequency chunks accumulated in TMEM, up to the
    80 x 80 limit); every sample of every instance against Tier A."""
    c = scw.Context(0)
    c.set_path(scw.SCW_PATH_TENSOR)
    try:
        g = np.random.default_rng(11)
        x = np.sort(g.uniform(-2, 5, 19))
        y = np.sort(g.uniform(-2, 5, 150))
        lays = [ragged_layer(U, Vn, J, np.complex64, seed=40 + i + J, ldV_pad=pad, with_c=(i % 2 == 0), with_dir=(i != 1))
                for i in range(n_inst)]
        zs = [np.linspace(-0.5 + 0.1 * i, 1.0, Fz) for i in range(n_inst)]
        Ls = [scw.Layer.from_numpy(l, "cuda") for l in lays]
        n0 = c.launch_count()
        Es = scw.scw_sweep_wavelengths(c, Ls, [dev(z) for z in zs], dev(x), dev(y))
        torch.cuda.synchronize()
        assert c.launch_count() - n0 == 3                               # twiddles, assembly (weights + fix-up inside), synthesis
        for lay, z, E in zip(lays, zs, Es):
            assert rel_err(E.cpu().numpy(), oracle.layer_grid(x=x, y=y, z=z, **lay)) <= 2e-4
        P = scw.scw_assemble_spectra(c, Ls[0], dev(zs[0]))
        E1 = scw.scw_synthesize_grid(c, U=U, Vn=Vn, X=lays[0]["X"], Y=lays[0]["Y"], P=P, x=dev(x), y=dev(y))
        torch.cuda.synchronize()
        assert float((E1 - Es[0]).abs().max() / Es[0].abs().max()) <= 2e-5   # other stream-K split, same values
    finally:
        c.close()


def test_custom_strides_interleaved_output(scw, ctx):
    """strides = (comp, z, y, x): write E as [Fz][Ny][Nx][3] (component fastest)."""
    lay = ragged_layer(5, 3, 20, np.complex64, seed=3)
    x = np.arange(24) * 3.0 / 24
    y = np.arange(10) * 4.5 / 10
    z = np.linspace(-0.4, 0.9, 4)
    L = scw.Layer.from_numpy(lay, "cuda")
    P = scw.scw_assemble_spectra(ctx, L, dev(z))
    out = torch.zeros((4, 10, 24, 3), dtype=torch.complex64, device="cuda")
    scw.scw_synthesize_grid(ctx, U=5, Vn=3, X=3.0, Y=4.5, P=P, x=dev(x), y=dev(y), out=out,
                            strides=(1, 10 * 24 * 3, 24 * 3, 3))
    planar = scw.scw_synthesize_grid(ctx, U=5, Vn=3, X=3.0, Y=4.5, P=P, x=dev(x), y=dev(y))
    torch.cuda.synchronize()
    assert torch.equal(out.permute(0, 3, 1, 2), planar)
    assert rel_err(planar.cpu().numpy(), oracle.layer_grid(x=x, y=y, z=z, **lay)) <= 2e-4


def test_empty_inputs_are_noops(scw, ctx):
    lay = ragged_layer(3, 3, 36, np.complex64, seed=1)
    L = scw.Layer.from_numpy(lay, "cuda")
    empty = torch.empty(0, dtype=torch.float64, device="cuda")
    n0 = ctx.launch_count()
    P = scw.scw_assemble_spectra(ctx, L, empty)
    assert P.shape == (0, 27)
    E = scw.scw_synthesize_grid(ctx, U=3, Vn=3, X=3.0, Y=4.5, P=P, x=dev(np.arange(4.0)), y=dev(np.arange(5.0)))
    assert E.shape == (0, 3, 5, 4)
    pts = scw.scw_eval_points(ctx, L, torch.empty((0, 3), dtype=torch.float64, device="cuda"))
    assert pts.shape == (0, 3)
    assert scw.scw_sweep_wavelengths(ctx, [], [], dev(np.arange(4.0)), dev(np.arange(5.0))) == []
    assert ctx.launch_count() == n0                                  # nothing was launched


def test_error_codes_and_nothing_written(scw, ctx):
    from paper_2404_07293_b200 import binding as b
    lay = ragged_layer(3, 3, 36, np.complex64, seed=2)
    L = scw.Layer.from_numpy(lay, "cuda")
    z = dev(np.linspace(-0.4, 0.9, 4))
    P = torch.full((4, 27), 5.0, dtype=torch.complex64, device="cuda")
    lib = ctx.L
    need = ctypes.c_size_t()

    def call(st, Fz=4, zp=z, Pp=P, ldP=27):
        return lib.scw_assemble_spectra(ctx._h, ctypes.byref(st), Fz, b._p(zp), b._p(Pp), ldP)

    ctx.reserve(1 << 20)
    st = L.struct(); st.lambda_ = 0.0
    assert call(st) == 5 and "lambda" in ctx.last_error()            # SCW_ERR_VALUE
    st = L.struct(); st.z_hi = st.z_lo - 1.0
    assert call(st) == 5
    st = L.struct(); st.X = float("nan")
    assert call(st) == 5
    st = L.struct(); st.dtype = 7
    assert call(st) == 3                                             # SCW_ERR_DTYPE
    st = L.struct(); st.ldV = 26
    assert call(st) == 2                                             # SCW_ERR_SHAPE
    st = L.struct(); st.J = 0
    assert call(st) == 2
    st = L.struct(); st.struct_size = 8
    assert call(st) == 2
    st = L.struct(); st.V = None
    assert call(st) == 1                                             # SCW_ERR_NULL
    st = L.struct(); st.V = L.V.data_ptr() + 4
    assert call(st) == 4                                             # SCW_ERR_ALIGN
    st = L.struct()
    assert call(st, ldP=26) == 2
    assert call(st, Fz=-1) == 2
    assert call(st, zp=None) == 1
    assert lib.scw_assemble_spectra(None, ctypes.byref(st), 4, b._p(z), b._p(P), 27) == 1
    # workspace too small: error, required size reported, nothing written
    lib.scw_assemble_workspace(ctx._h, ctypes.byref(st), 4, ctypes.byref(need))
    assert need.value > 0
    small = torch.empty(256, dtype=torch.uint8, device="cuda")
    assert lib.scw_set_workspace(ctx._h, b._p(small), 256) == 0
    assert call(st) == 6 and lib.scw_required_workspace(ctx._h) == need.value
    torch.cuda.synchronize()
    assert torch.all(P == 5.0)                                       # nothing was written by any failing call
    ctx._ws = None
    ctx.reserve(need.value)
    assert call(st) == 0
    torch.cuda.synchronize()
    assert not torch.all(P == 5.0)
    # misaligned workspace / unknown option
    assert lib.scw_set_workspace(ctx._h, ctypes.c_void_p(ctx._ws.data_ptr() + 8), 1024) == 4
    assert lib.scw_set_option(ctx._h, 99, 0) == 8
    # sweep with mismatching instances
    lay2 = ragged_layer(5, 3, 20, np.complex64, seed=3)
    with pytest.raises(scw.ScwError) as e:
        scw.scw_sweep_wavelengths(ctx, [L, scw.Layer.from_numpy(lay2, "cuda")], [z, z], dev(np.arange(4.0)),
                                  dev(np.arange(4.0)))
    assert e.value.status == 2
    # points: bad kind / N < 0
    m = b.scw_modes(); m.struct_size = ctypes.sizeof(b.scw_modes); m.kind = 5
    assert lib.scw_eval_points(ctx._h, ctypes.byref(m), 1, b._p(z), b._p(P)) == 2
    pw = scw.PlaneWaves.from_numpy(si.make_planewaves(si.CONFIGS[3]), "cuda").struct()
    assert lib.scw_eval_points(ctx._h, ctypes.byref(pw), -3, b._p(z), b._p(P)) == 2
    pw.lambda_ = -1.0
    assert lib.scw_eval_points(ctx._h, ctypes.byref(pw), 1, b._p(z), b._p(P)) == 5


def test_stream_and_launch_counter(scw):
    """Work is enqueued on the stream given at creation; the launch counter advances."""
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        c = scw.Context(0, stream=s)
        lay = ragged_layer(3, 3, 36, np.complex128, seed=4)
        z = dev(np.linspace(-0.4, 0.9, 2))
        x, y = np.arange(6) * 0.5, np.arange(4) * 1.125
        n0 = c.launch_count()
        E = scw.scw_sweep_wavelengths(c, [scw.Layer.from_numpy(lay, "cuda")], [z], dev(x), dev(y))[0]
        assert c.launch_count() > n0
        s.synchronize()
    assert rel_err(E.cpu().numpy(), oracle.layer_grid(x=x, y=y, z=np.linspace(-0.4, 0.9, 2), **lay)) <= 1e-10
    c.close()


def test_more_tiles_than_sms_and_more_instances_than_a_group(scw):
    """Tensor path at its scheduling edges: 14 x 11 = 154 output tiles (two synthesis launches over the tile pairs, each
    pair's planes handed out dynamically), and 70 instances (two groups of the grouped sweep); every sample against the
    factored fp64 reference (Tier B, itself pinned to Tier A)."""
    c = scw.Context(0)
    c.set_path(scw.SCW_PATH_TENSOR)
    try:
        g = np.random.default_rng(23)
        lay = ragged_layer(6, 5, 64, np.complex64, seed=77)
        x = np.sort(g.uniform(-3, 9, 1700))
        y = np.sort(g.uniform(-3, 9, 1300))
        z = np.array([0.1, 0.7])
        E = scw.scw_sweep_wavelengths(c, [scw.Layer.from_numpy(lay, "cuda")], [dev(z)], dev(x), dev(y))[0]
        torch.cuda.synchronize()
        assert rel_err(E.cpu().numpy(), oracle.tier_b_grid(x=x, y=y, z=z, **lay)) <= 2e-4
        lays = [ragged_layer(4, 3, 40, np.complex64, seed=200 + i, with_c=(i % 3 != 0)) for i in range(70)]
        xs, ys = np.linspace(0, 3, 33), np.linspace(0, 4.5, 140)
        zs = [np.array([0.0, 0.3 + 0.01 * i, 0.9]) for i in range(70)]
        Es = scw.scw_sweep_wavelengths(c, [scw.Layer.from_numpy(l, "cuda") for l in lays], [dev(v) for v in zs], dev(xs), dev(ys))
        I = scw.scw_sweep_intensity(c, [scw.Layer.from_numpy(l, "cuda") for l in lays], [dev(v) for v in zs], dev(xs), dev(ys))
        torch.cuda.synchronize()
        for i in (0, 1, 63, 64, 69):
            ref = oracle.tier_b_grid(x=xs, y=ys, z=zs[i], **lays[i])
            assert rel_err(Es[i].cpu().numpy(), ref) <= 2e-4
            Iref = oracle.intensity(ref)
            assert np.abs(I[i].cpu().numpy() - Iref).max() / Iref.max() <= 4e-4
    finally:
        c.close()


def test_many_tiles_few_planes_twice_into_one_workspace(scw, ctx):
    """3 x 3 frequencies, one z plane, 3072 x 3072 grid = 576 output tiles: more plane counters than threads of the
    spectrum-image kernel (they must all be reset), run twice into the same workspace; NaN sentinels must all be
    overwritten and a seeded subset must match Tier A."""
    lay = ragged_layer(3, 3, 36, np.complex64, seed=77)
    N = 3072
    x = np.arange(N) * (3.0 / N)
    y = np.arange(N) * (4.5 / N)
    z = np.array([0.2])
    L = scw.Layer.from_numpy(lay, "cuda")
    P = scw.scw_assemble_spectra(ctx, L, dev(z))
    dx, dy = dev(x), dev(y)
    g = np.random.default_rng(9)
    iy, ix = g.integers(0, N, 400), g.integers(0, N, 400)
    xyz = np.column_stack([x[ix], y[iy], np.full(400, z[0])])
    ref = oracle.layer_samples(xyz=xyz, **lay)
    for _ in range(2):
        E = torch.full((1, 3, N, N), float("nan"), dtype=torch.complex64, device="cuda")
        scw.scw_synthesize_grid(ctx, U=3, Vn=3, X=lay["X"], Y=lay["Y"], P=P, x=dx, y=dy, out=E)
        torch.cuda.synchronize()
        assert not bool(torch.isnan(E.real).any())
        got = E[0][:, torch.from_numpy(iy).cuda(), torch.from_numpy(ix).cuda()].T.cpu().numpy()
        assert np.abs(got - ref).max() / np.abs(ref).max() <= 2e-4
        del E


def test_grouped_sweep_with_an_8_byte_aligned_V(scw, ctx):
    """Instance 1 of a sweep holds V at an address that is only 8-byte aligned (a view one element into a buffer): the
    TMA assembly cannot take it, so the whole sweep must drop to the per-instance path (CUDA-core assembly for that
    instance) instead of failing in cuTensorMapEncodeTiled."""
    lays = [ragged_layer(5, 5, 100, np.complex64, seed=90 + i) for i in range(3)]
    x = np.arange(20) * 3.0 / 20
    y = np.arange(18) * 4.5 / 18
    z = np.linspace(-0.3, 0.8, 4)
    Ls = [scw.Layer.from_numpy(l, "cuda") for l in lays]
    J, ld = Ls[1].V.shape
    buf = torch.zeros(J * ld + 1, dtype=torch.complex64, device="cuda")
    buf[1:] = Ls[1].V.reshape(-1)
    Ls[1].V = buf[1:].view(J, ld)
    assert Ls[1].V.data_ptr() % 16 == 8
    Es = scw.scw_sweep_wavelengths(ctx, Ls, [dev(z)] * 3, dev(x), dev(y))
    torch.cuda.synchronize()
    for lay, E in zip(lays, Es):
        assert rel_err(E.cpu().numpy(), oracle.layer_grid(x=x, y=y, z=z, **lay)) <= 2e-4


def test_last_kernels_tells_which_path_ran(scw, ctx):
    """SCW_PATH_AUTO drops to the CUDA-core kernels for shapes the tensor-core kernels do not take; scw_last_kernels makes
    that visible: complex64 with 96 frequencies along u (> 80) synthesises on CUDA cores, a sweep whose instances differ in J
    is cut into runs of equal shape (one assembly + one synthesis launch each), a regular one takes tc_assemble + tc_synth."""
    lay = ragged_layer(5, 5, 100, np.complex64, seed=7)
    x, y, z = np.arange(20) * 0.15, np.arange(18) * 0.25, np.linspace(-0.3, 0.8, 4)
    L = scw.Layer.from_numpy(lay, "cuda")
    scw.scw_sweep_wavelengths(ctx, [L], [dev(z)], dev(x), dev(y))
    assert {"tc_assemble", "tc_synth"} <= set(ctx.last_kernels()) and not any(k.startswith("simt") for k in ctx.last_kernels())
    wide = ragged_layer(96, 2, 64, np.complex64, seed=8)
    scw.scw_sweep_wavelengths(ctx, [scw.Layer.from_numpy(wide, "cuda")], [dev(z)], dev(x), dev(y))
    assert "simt_synth_b" in ctx.last_kernels() and "tc_synth" not in ctx.last_kernels()
    lay2 = ragged_layer(5, 5, 132, np.complex64, seed=9)
    n0 = ctx.launch_count()
    scw.scw_sweep_wavelengths(ctx, [L, scw.Layer.from_numpy(lay2, "cuda")], [dev(z), dev(z)], dev(x), dev(y))
    torch.cuda.synchronize()
    assert ctx.launch_count() - n0 == 5                                      # twiddles + two runs (J differs) x (assembly, synthesis)
    assert not any(k.startswith("simt") for k in ctx.last_kernels())


def test_twiddle_cache_and_calibration(scw):
    """SCW_OPT_CACHE: consecutive sweeps reuse the twiddle tables, the clean control block and the zeroed image padding (two
    launches instead of three); results stay those of the oracle; scw_invalidate_cache picks up coordinates changed in
    place; a different call in between drops the cache; scw_calibrate changes the split, not the values."""
    c = scw.Context(0)
    try:
        c.set_cache(True)
        lays = [ragged_layer(9, 7, 252, np.complex64, seed=60 + i) for i in range(3)]
        x = np.arange(150) * 3.0 / 150
        y = np.arange(140) * 4.5 / 140
        z = np.linspace(-0.2, 0.8, 5)
        Ls = [scw.Layer.from_numpy(l, "cuda") for l in lays]
        dx, dy, dzs = dev(x), dev(y), [dev(z)] * 3
        refs = [oracle.tier_b_grid(x=x, y=y, z=z, **l) for l in lays]
        n0 = c.launch_count()
        E1 = [e.clone() for e in scw.scw_sweep_wavelengths(c, Ls, dzs, dx, dy)]
        n1 = c.launch_count()
        E2 = scw.scw_sweep_wavelengths(c, Ls, dzs, dx, dy)
        n2 = c.launch_count()
        torch.cuda.synchronize()
        assert n1 - n0 == 3 and n2 - n1 == 2                               # the second call skips the twiddle kernel
        for a, b, r in zip(E1, E2, refs):
            assert torch.equal(a, b)
            assert rel_err(b.cpu().numpy(), r) <= 2e-4
        I = scw.scw_sweep_intensity(c, Ls, dzs, dx, dy)                     # same workspace layout family: still cached
        torch.cuda.synchronize()
        assert np.abs(I[0].cpu().numpy() - oracle.intensity(refs[0])).max() / oracle.intensity(refs[0]).max() <= 4e-4
        # coordinates changed in place: stale until invalidated
        dx.mul_(0.5)
        c.invalidate_cache()
        E3 = scw.scw_sweep_wavelengths(c, Ls, dzs, dx, dy)
        torch.cuda.synchronize()
        assert rel_err(E3[1].cpu().numpy(), oracle.tier_b_grid(x=0.5 * x, y=y, z=z, **lays[1])) <= 2e-4
        # another kind of call carves the workspace differently: the next sweep must not trust the cache
        scw.scw_assemble_spectra(c, Ls[0], dzs[0])
        n3 = c.launch_count()
        E4 = scw.scw_sweep_wavelengths(c, Ls, dzs, dx, dy)
        torch.cuda.synchronize()
        assert c.launch_count() - n3 == 3 and torch.equal(E4[2], E3[2])
        # calibration: same values up to the summation order of the stream-K split
        E5 = scw.scw_calibrate(c, Ls, dzs, dx, dy, reps=2)
        E6 = scw.scw_sweep_wavelengths(c, Ls, dzs, dx, dy)
        torch.cuda.synchronize()
        for a, b in zip(E5, E6):
            assert float((a - E3[0].new_tensor(0) - b).abs().max()) == 0.0     # same split after calibration: identical
        assert float((E6[0] - E3[0]).abs().max() / E3[0].abs().max()) <= 2e-5
        assert len(c.assembly_timeline()) >= 1
    finally:
        c.close()


def test_sweep_captured_in_a_cuda_graph(scw):
    """The library only enqueues work on the ctx stream (no synchronisation, no allocation): a cached sweep can be captured
    into a CUDA graph and replayed; the replay writes what the plain call writes."""
    s = torch.cuda.Stream()
    c = scw.Context(0, stream=s)
    try:
        c.set_cache(True)
        lays = [ragged_layer(9, 7, 252, np.complex64, seed=90 + i) for i in range(3)]
        Ls = [scw.Layer.from_numpy(l, "cuda") for l in lays]
        x, y, z = dev(np.arange(150) * 3.0 / 150), dev(np.arange(140) * 4.5 / 140), dev(np.linspace(-0.2, 0.8, 5))
        out = [torch.empty((5, 3, 140, 150), dtype=torch.complex64, device="cuda") for _ in Ls]
        with torch.cuda.stream(s):
            for _ in range(2):                                              # warm: workspace sized, twiddles cached
                scw.scw_sweep_wavelengths(c, Ls, [z] * 3, x, y, out=out)
            s.synchronize()
            ref = [o.clone() for o in out]
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=s):
                scw.scw_sweep_wavelengths(c, Ls, [z] * 3, x, y, out=out)
            for o in out:
                o.zero_()
            g.replay()
            s.synchronize()
        for a, b, l in zip(out, ref, lays):
            assert torch.equal(a, b)
            assert rel_err(a.cpu().numpy(), oracle.tier_b_grid(x=x.cpu().numpy(), y=y.cpu().numpy(), z=z.cpu().numpy(), **l)) <= 2e-4
    finally:
        c.close()


def test_measure_peak_units_and_errors(scw, ctx):
    """scw_measure_peak: every unit returns a rate in a sane range for a B200 (an order of magnitude either side of the
    nominal figures), the sin + cos + ex2 mix runs on the same pipe as the ex2 chain, unknown units are refused."""
    from paper_2404_07293_b200 import binding as b
    peaks = ctx.measure_peaks(reps=2, hbm_bytes=1 << 28)
    assert set(peaks) == set(b.SCW_PEAKS)
    assert 10.0 < peaks["fp64_dmma_tflops"] < 100.0 and 20.0 < peaks["fp32_fma_tflops"] < 200.0
    assert 1000.0 < peaks["mufu_gops"] < 10000.0
    assert 0.8 < peaks["mufu_sincosex2_gops"] / peaks["mufu_gops"] < 1.2
    for k in ("hbm_read_gbs", "hbm_write_gbs", "hbm_write_tma_gbs"):
        assert 2000.0 < peaks[k] < 12000.0, (k, peaks[k])
    buf = torch.empty(1 << 20, dtype=torch.uint8, device="cuda")
    v = ctypes.c_double()
    rc = ctx.L.scw_measure_peak(ctx._h, 99, ctypes.c_void_p(buf.data_ptr()), buf.numel(), 1, ctypes.byref(v))
    assert rc == 5 and v.value == 0.0                                        # SCW_ERR_VALUE
    rc = ctx.L.scw_measure_peak(ctx._h, 2, None, 0, 1, ctypes.byref(v))
    assert rc == 1                                                           # SCW_ERR_NULL


def test_kernel_timeline_of_the_sweep_kernels(scw):
    """scw_profile_timeline: every tensor-core sweep launch leaves its exit time on the device clock; entries come oldest
    first, alternate assembly / synthesis, never decrease, and a call that is not a sweep leaves them alone."""
    c = scw.Context(0)
    try:
        assert c.kernel_timeline() == []
        c.set_cache(True)
        lay = ragged_layer(9, 7, 252, np.complex64, seed=77)
        L = scw.Layer.from_numpy(lay, "cuda")
        x, y, z = dev(np.arange(150) * 3.0 / 150), dev(np.arange(140) * 4.5 / 140), dev(np.linspace(0.1, 0.7, 5))
        for _ in range(4):
            scw.scw_sweep_wavelengths(c, [L, L], [z, z], x, y)
        tl = c.kernel_timeline()
        assert [k for _, k in tl] == ["tc_assemble", "tc_synth"] * 4
        t = [ns for ns, _ in tl]
        assert all(b > a for a, b in zip(t, t[1:])) and t[-1] - t[0] < 1e9      # strictly later, all within a second
        assert c.kernel_timeline(3) == tl[-3:]
        scw.scw_assemble_spectra(c, L, z)                                     # its own launch is not part of the ring's order
        for _ in range(70):                                                   # more launches than the ring holds
            scw.scw_sweep_wavelengths(c, [L, L], [z, z], x, y)
        tl = c.kernel_timeline()
        assert len(tl) == 128 and [k for _, k in tl] == ["tc_assemble", "tc_synth"] * 64
        t = [ns for ns, _ in tl]
        assert all(b > a for a, b in zip(t, t[1:]))
    finally:
        c.close()


def test_sweep_with_mixed_shapes_runs_grouped(scw, ctx):
    """Instances that differ in J and in Fz: consecutive instances of equal shape form a run (one assembly + one synthesis
    launch per run, all on the tensor-core kernels); every sample of every instance against Tier B."""
    shapes = [(100, 4), (100, 4), (132, 4), (132, 7), (132, 7), (100, 4)]
    lays = [ragged_layer(5, 5, J, np.complex64, seed=120 + i) for i, (J, _) in enumerate(shapes)]
    zs = [np.linspace(-0.3, 0.8, fz) for _, fz in shapes]
    x, y = np.arange(150) * 3.0 / 150, np.arange(40) * 4.5 / 40
    Ls = [scw.Layer.from_numpy(l, "cuda") for l in lays]
    n0 = ctx.launch_count()
    Es = scw.scw_sweep_wavelengths(ctx, Ls, [dev(z) for z in zs], dev(x), dev(y))
    S = scw.scw_sweep_detector(ctx, Ls, [dev(z) for z in zs], dev(x), dev(y), window=(3, 140, 2, 33), want_I=False)[1]
    torch.cuda.synchronize()
    for lay, z, E, s in zip(lays, zs, Es, S):
        ref = oracle.tier_b_grid(x=x, y=y, z=z, **lay)
        assert rel_err(E.cpu().numpy(), ref) <= 2e-4
        sref = oracle.window_sum(oracle.intensity(ref), (3, 140, 2, 33))
        assert np.abs(s.cpu().numpy() - sref).max() / sref.max() <= 4e-4
    assert not any(k.startswith("simt") for k in ctx.last_kernels())


def test_sweep_small_run_before_a_large_one(scw):
    """Runs of different size share one assembly scratch, and each run keeps its per-CTA timers and weight images right
    behind its own tile counters: a 1-instance run followed by a 6-instance run (2 m-tiles each) must not leave the
    larger run's counters dirty (its fix-up would be skipped and the spectrum images stay stale).  Every sample against
    Tier B; then the same with SCW_OPT_CACHE on and the inputs exchanged between two calls (large run first, so that the
    LAST run of the call is the small one and the next call may not trust the largest run's control block)."""
    x, y = np.arange(150) * 3.0 / 150, np.arange(40) * 4.5 / 40
    z = np.linspace(-0.3, 0.8, 4)
    dx, dy = dev(x), dev(y)

    def check(c, shapes, seed0):
        lays = [ragged_layer(9, 7, J, np.complex64, seed=seed0 + i) for i, J in enumerate(shapes)]
        Es = scw.scw_sweep_wavelengths(c, [scw.Layer.from_numpy(l, "cuda") for l in lays], [dev(z)] * len(lays), dx, dy)
        torch.cuda.synchronize()
        assert not any(k.startswith("simt") for k in c.last_kernels())
        for i, (lay, E) in enumerate(zip(lays, Es)):
            assert rel_err(E.cpu().numpy(), oracle.tier_b_grid(x=x, y=y, z=z, **lay)) <= 2e-4, i

    c = scw.Context(0)
    try:
        check(c, [100] + [132] * 6, 300)
        check(c, [100, 100] + [132] * 3 + [100] + [132] * 5, 320)
        c.set_cache(True)
        check(c, [132] * 6 + [100] * 2, 340)
        check(c, [132] * 6 + [100] * 2, 360)           # same shapes, new inputs: stale images would be call 1's fields
        check(c, [100] + [132] * 6, 380)
    finally:
        c.close()


def test_cache_survives_alternating_paths_and_layouts(scw):
    """SCW_OPT_CACHE on: a grouped tensor-core sweep, then a sweep that carves the same workspace differently (the
    CUDA-core path; a sweep with an instance the grouped kernels cannot take, here J = 1), then the grouped sweep again.
    The middle sweeps overwrite the grouped layout's control block and image padding: the last sweep must clear them
    again instead of trusting the cache.  Every sample of every sweep against Tier B."""
    x, y = np.arange(150) * 3.0 / 150, np.arange(140) * 4.5 / 140
    z = np.linspace(-0.2, 0.8, 5)
    dx, dy = dev(x), dev(y)

    def sweep(c, lays):
        Es = scw.scw_sweep_wavelengths(c, [scw.Layer.from_numpy(l, "cuda") for l in lays], [dev(z)] * len(lays), dx, dy)
        torch.cuda.synchronize()
        for i, (lay, E) in enumerate(zip(lays, Es)):
            assert rel_err(E.cpu().numpy(), oracle.tier_b_grid(x=x, y=y, z=z, **lay)) <= 2e-4, i
        return c.last_kernels()

    c = scw.Context(0)
    try:
        c.set_cache(True)
        grouped = [ragged_layer(9, 7, 252, np.complex64, seed=400 + i) for i in range(4)]
        assert not any(k.startswith("simt") for k in sweep(c, grouped))
        c.set_path(scw.SCW_PATH_SIMT)
        assert not any(k.startswith("tc_") for k in sweep(c, grouped))
        c.set_path(scw.SCW_PATH_AUTO)
        assert not any(k.startswith("simt") for k in sweep(c, grouped))
        # per-instance layout in the middle: one instance with a single mode
        mixed = [ragged_layer(9, 7, 252, np.complex64, seed=410), ragged_layer(9, 7, 1, np.complex64, seed=411),
                 ragged_layer(9, 7, 252, np.complex64, seed=412)]
        sweep(c, mixed)
        assert not any(k.startswith("simt") for k in sweep(c, grouped))
        sweep(c, mixed)
        sweep(c, [ragged_layer(9, 7, 252, np.complex64, seed=420 + i) for i in range(4)])
    finally:
        c.close()


def test_profile_readers_forget_a_replaced_workspace(scw):
    """The per-CTA timers and the timeline ring of a sweep live in the workspace.  After the caller registers another
    workspace (the old one may be freed) the readers must report 'nothing recorded' instead of copying from the old
    address; the next sweep records again."""
    c = scw.Context(0)
    try:
        lays = [ragged_layer(9, 7, 252, np.complex64, seed=500 + i) for i in range(2)]
        x, y, z = np.arange(150) * 3.0 / 150, np.arange(140) * 4.5 / 140, np.linspace(-0.2, 0.8, 5)
        Ls = [scw.Layer.from_numpy(l, "cuda") for l in lays]
        scw.scw_sweep_wavelengths(c, Ls, [dev(z)] * 2, dev(x), dev(y))
        assert len(c.assembly_timeline()) >= 1 and len(c.kernel_timeline()) == 2
        c.reserve(c.workspace_bytes() + (1 << 20))               # a new, larger buffer: scw_set_workspace
        torch.cuda.empty_cache()                                 # the old one really goes back to the driver
        assert c.assembly_timeline() == [] and c.kernel_timeline() == []
        scw.scw_sweep_wavelengths(c, Ls, [dev(z)] * 2, dev(x), dev(y))
        assert len(c.assembly_timeline()) >= 1 and len(c.kernel_timeline()) == 2
    finally:
        c.close()


@pytest.mark.parametrize("Nx,Ny", [(1, 150), (150, 1), (1, 1)])
@pytest.mark.parametrize("U,Vn,J,Fz", [(7, 9, 250, 20), (45, 50, 64, 4)])
def test_xz_and_yz_planes(scw, Nx, Ny, U, Vn, J, Fz):
    """x-z and y-z planes ('The same goes for x-z and y-z planes'): the separable synthesis with ONE
    coordinate along an axis -- a 1-wide axis through the 128 x 128 output tiles of the forced tcgen05 path (complex64),
    through the DMMA path (complex128) and through the fused detector epilogue; every sample against Tier A."""
    g = np.random.default_rng(1000 * Nx + Ny)
    x = np.sort(g.uniform(-2, 5, Nx))
    y = np.sort(g.uniform(-2, 5, Ny))
    z = np.linspace(-0.4, 0.9, Fz)
    for dtype, tol, path in ((np.complex64, 2e-4, "tensor"), (np.complex128, 1e-10, "auto")):
        lay = ragged_layer(U, Vn, J, dtype, seed=70 + U + Nx)
        ref = oracle.layer_grid(x=x, y=y, z=z, **lay)
        c = scw.Context(0)
        try:
            if path == "tensor":
                c.set_path(scw.SCW_PATH_TENSOR)
            L = scw.Layer.from_numpy(lay, "cuda")
            E = scw.scw_sweep_wavelengths(c, [L], [dev(z)], dev(x), dev(y))[0]
            torch.cuda.synchronize()
            assert E.shape == (Fz, 3, Ny, Nx)
            assert rel_err(E.cpu().numpy(), ref) <= tol
            kinds = c.last_kernels()
            assert any(k.startswith("tc_") for k in kinds) if path == "tensor" else any(k.startswith("dmma") for k in kinds)
            P = scw.scw_assemble_spectra(c, L, dev(z))
            E2 = scw.scw_synthesize_grid(c, U=U, Vn=Vn, X=lay["X"], Y=lay["Y"], P=P, x=dev(x), y=dev(y))
            torch.cuda.synchronize()
            assert rel_err(E2.cpu().numpy(), ref) <= tol
            I, S = scw.scw_sweep_detector(c, [L], [dev(z)], dev(x), dev(y))
            torch.cuda.synchronize()
            Iref = oracle.intensity(ref)
            assert np.abs(I[0].cpu().numpy() - Iref).max() / Iref.max() <= 2 * tol
            sref = oracle.window_sum(Iref, (0, Nx, 0, Ny))
            assert np.abs(S[0].cpu().numpy() - sref).max() / sref.max() <= 2 * tol
        finally:
            c.close()

"""GPU parity of the exterior field (eq. 9-10) against the eq. 9-10 oracle, through the C ABI."""
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


def ext_z(ext, n, lam):
    """n planes in the half-space, from the interface outwards (the interface itself included)."""
    d = np.linspace(0.0, 3.0 * lam, n)
    return ext["z_face"] - d if ext["side"] == oracle.SIDE_ABOVE else ext["z_face"] + d


@pytest.mark.parametrize("dtype,tol", [(np.complex128, 1e-10), (np.complex64, 2e-4)])
@pytest.mark.parametrize("side", [0, 1])
def test_config0_exterior_grid_and_points(scw, ctx, side, dtype, tol):
    """Config 0's half-spaces (n = 1.0 above, 1.5 below): every sample of a 64 x 64 x 8 grid through
    scw_exterior_spectra + scw_synthesize_grid, and the same samples through scw_exterior_points."""
    cfg = si.CONFIGS[0]
    ext = si.make_exterior(cfg, side, dtype=dtype)
    x, y, _ = si.grid_coords(cfg, 0)
    z = ext_z(ext, 8, ext["lam"])
    ref = oracle.exterior_grid(x=x, y=y, z=z, **ext)
    X = scw.Exterior.from_numpy(ext, "cuda")
    P = scw.scw_exterior_spectra(ctx, X, dev(z))
    E = scw.scw_synthesize_grid(ctx, U=ext["U"], Vn=ext["Vn"], X=ext["X"], Y=ext["Y"], P=P, x=dev(x), y=dev(y))
    xyz = oracle.grid_points(x, y, z)
    Ep = scw.scw_exterior_points(ctx, X, dev(xyz))
    torch.cuda.synchronize()
    scale = np.abs(ref).max()
    assert np.abs(E.cpu().numpy() - ref).max() / scale <= tol
    got = Ep.cpu().numpy().reshape(len(z), len(y), len(x), 3).transpose(0, 3, 1, 2)
    assert np.abs(got - ref).max() / scale <= tol


@pytest.mark.parametrize("side", [0, 1])
def test_config1_shape_exterior_full_size_c64(scw, ctx, side):
    """33 x 33 orders on the 256 x 256 x 16 grid (tcgen05 synthesis fed by eq. 9 spectra): seeded sample subset."""
    cfg = si.CONFIGS[1]
    ext = si.make_exterior(cfg, side, dtype=np.complex64)
    x, y, _ = si.grid_coords(cfg, 0)
    z = ext_z(ext, 16, ext["lam"])
    X = scw.Exterior.from_numpy(ext, "cuda")
    P = scw.scw_exterior_spectra(ctx, X, dev(z))
    E = scw.scw_synthesize_grid(ctx, U=cfg.U, Vn=cfg.Vn, X=ext["X"], Y=ext["Y"], P=P, x=dev(x), y=dev(y))
    torch.cuda.synchronize()
    idx = si.sample_subset(cfg, len(z) * cfg.Ny * cfg.Nx, 6000, layer=side)
    iz, iy, ix = np.unravel_index(idx, (len(z), cfg.Ny, cfg.Nx))
    ref = oracle.exterior_samples(xyz=np.column_stack([x[ix], y[iy], z[iz]]), **ext)
    got = E.cpu().numpy()[iz, :, iy, ix]
    assert np.abs(got - ref).max() / np.abs(ref).max() <= 2e-4
    # scattered points (not on the grid) through the direct sum
    g = np.random.default_rng(17 + side)
    xyz = np.column_stack([g.uniform(0, cfg.L, 3001), g.uniform(0, cfg.L, 3001), ext_z(ext, 3001, ext["lam"])])
    Ep = scw.scw_exterior_points(ctx, X, dev(xyz))
    torch.cuda.synchronize()
    refp = oracle.exterior_samples(xyz=xyz, **ext)
    assert np.abs(Ep.cpu().numpy() - refp).max() / np.abs(refp).max() <= 2e-4


def test_exterior_edges_and_errors(scw, ctx):
    """No incident wave, ragged frequency counts, padded ldP, empty calls, argument errors (nothing written)."""
    ext = dict(side=0, U=4, Vn=3, X=3.0, Y=5.0, lam=0.8, n=1.2, z_face=0.5,
               p_face=(np.arange(36).reshape(12, 3) * (0.1 - 0.05j)).astype(np.complex128))
    z = np.array([0.5, 0.1, -1.0])
    X = scw.Exterior.from_numpy(ext, "cuda")
    Pbuf = torch.full((3, 36 + 4), 7.0, dtype=torch.complex128, device="cuda")
    scw.scw_exterior_spectra(ctx, X, dev(z), out=Pbuf)
    xs, ys = np.array([0.0, 0.7, 2.9]), np.array([1.0, 4.4])
    E = scw.scw_synthesize_grid(ctx, U=4, Vn=3, X=3.0, Y=5.0, P=Pbuf, x=dev(xs), y=dev(ys))
    torch.cuda.synchronize()
    assert torch.all(Pbuf[:, 36:] == 7.0)
    ref = oracle.exterior_grid(x=xs, y=ys, z=z, **ext)
    assert np.abs(E.cpu().numpy() - ref).max() / np.abs(ref).max() <= 1e-10
    assert scw.scw_exterior_points(ctx, X, torch.empty((0, 3), dtype=torch.float64, device="cuda")).shape == (0, 3)
    bad = scw.Exterior.from_numpy(dict(ext, side=1, p_inc=ext["p_face"]), "cuda")       # incident wave below the sample
    with pytest.raises(scw.ScwError) as e:
        scw.scw_exterior_spectra(ctx, bad, dev(z))
    assert e.value.status == 5
    with pytest.raises(scw.ScwError) as e:
        scw.scw_exterior_spectra(ctx, scw.Exterior.from_numpy(dict(ext, lam=-1.0), "cuda"), dev(z))
    assert e.value.status == 5


@pytest.mark.parametrize("dtype,tol", [(np.complex128, 1e-10), (np.complex64, 2e-4)])
@pytest.mark.parametrize("side", [0, 1])
@pytest.mark.parametrize("U,Vn", [(9, 9), (45, 12)])
def test_exterior_grid_one_call(scw, dtype, tol, side, U, Vn):
    """scw_exterior_grid (eq. 9 straight into the synthesis operand for complex64; spectra + synthesis for complex128):
    every sample against the eq. 9-10 oracle, ragged grid, two frequency chunks along u, custom strides, twice with the
    twiddle cache on (the second call reuses the tables), then with other planes."""
    cfg = si.Config(6, "exterior grid", U, Vn, 8.0, (1.0,), 1, 1, 0, 0, (dtype,))
    ext = si.make_exterior(cfg, side, dtype=dtype)
    g = np.random.default_rng(U + side)
    x, y = np.sort(g.uniform(0, 8, 150)), np.sort(g.uniform(0, 8, 37))
    z = ext_z(ext, 5, ext["lam"])
    ref = oracle.exterior_grid(x=x, y=y, z=z, **ext)
    c = scw.Context(0)
    try:
        c.set_cache(True)
        X = scw.Exterior.from_numpy(ext, "cuda")
        dx, dy = dev(x), dev(y)
        n0 = c.launch_count()
        E1 = scw.scw_exterior_grid(c, X, dev(z), dx, dy).clone()
        n1 = c.launch_count()
        out = torch.zeros((5, 37, 150, 3), dtype=E1.dtype, device="cuda")             # [z][y][x][comp]
        scw.scw_exterior_grid(c, X, dev(z), dx, dy, out=out, strides=(1, 37 * 150 * 3, 150 * 3, 3))
        n2 = c.launch_count()
        z2 = ext_z(ext, 3, 0.5 * ext["lam"])
        E3 = scw.scw_exterior_grid(c, X, dev(z2), dx, dy)
        torch.cuda.synchronize()
        scale = np.abs(ref).max()
        assert np.abs(E1.cpu().numpy() - ref).max() / scale <= tol
        assert torch.equal(out.permute(0, 3, 1, 2), E1)
        assert np.abs(E3.cpu().numpy() - oracle.exterior_grid(x=x, y=y, z=z2, **ext)).max() / scale <= tol
        if dtype == np.complex64:
            assert n1 - n0 == 3 and n2 - n1 == 2                   # twiddles + images + synthesis, then cached twiddles
            assert "tc_synth" in c.last_kernels()
    finally:
        c.close()

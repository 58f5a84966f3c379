"""Detector intensity I = sum_comp |E_comp|^2: oracle pins (CPU) and GPU parity through the C ABI.

Tolerance: dI = 2 Re(E* dE) summed over components, so a field error of eps * max|E| gives at most 2 eps * max I:
4e-4 of max I for complex64 (field bar 2e-4), 2e-10 for complex128.
"""
import numpy as np
import pytest

import oracle
import scw_inputs as si


def test_intensity_closed_form_and_parseval():
    """Single mode, single frequency: I = sum_comp |c V|^2 exp(-2 k Im(gamma) dz), flat in x, y; and Parseval:
    sum_xy I = Nx Ny sum_comp sum_m |P|^2 on a grid spanning one period (Nx >= U, Ny >= V)."""
    cfg = si.CONFIGS[0]
    lay = si.make_layer(cfg, dtype=np.complex128)
    U, Vn, M = lay["U"], lay["Vn"], lay["U"] * lay["Vn"]
    j, m = 6, 40                                                  # a "+" mode: referenced at z_lo
    V1 = np.zeros_like(lay["V"])
    for comp in range(3):
        V1[j, comp * M + m] = lay["V"][j, comp * M + m]
    one = dict(lay, V=V1)
    x, y, z = np.array([0.3, 5.1]), np.array([1.7]), np.array([0.4, 1.9])
    I = oracle.intensity(oracle.layer_grid(x=x, y=y, z=z, **one))
    amp2 = sum(abs(lay["c"][j] * lay["V"][j, comp * M + m]) ** 2 for comp in range(3))
    ref = amp2 * np.exp(-2 * (2 * np.pi / lay["lam"]) * lay["gamma"][j].imag * (z - lay["z_lo"]))
    assert lay["dir"][j] > 0 and np.allclose(I, ref[:, None, None] * np.ones((2, 1, 2)), rtol=1e-12)
    xg, yg, zg = si.grid_coords(cfg, 0, planes=2, Nx=16, Ny=12)
    If = oracle.intensity(oracle.tier_b_grid(x=xg, y=yg, z=zg, **lay))
    P = oracle.tier_b_spectra(z=zg, **lay)
    assert np.allclose(If.sum(axis=(1, 2)), 16 * 12 * (np.abs(P) ** 2).sum(axis=0), rtol=1e-11)


# ------------------------------------------------------------------------------------------------ GPU
@pytest.fixture(scope="module")
def scw():
    import paper_2404_07293_b200 as m
    m.lib()
    return m


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.gpu
@pytest.mark.parametrize("dtype,tol", [(np.complex128, 2e-10), (np.complex64, 4e-4)])
@pytest.mark.parametrize("path", ["auto", "tensor"])
def test_config0_intensity_every_sample(scw, dtype, tol, path):
    """Config 0: general path (complex128: DMMA + reduction kernel; complex64 auto: tcgen05 epilogue) against Tier A."""
    import torch
    cfg = si.CONFIGS[0]
    lay = si.make_layer(cfg, dtype=dtype)
    x, y, z = si.grid_coords(cfg, 0, planes=5, Nx=40, Ny=24)
    ref = oracle.intensity(oracle.layer_grid(x=x, y=y, z=z, **lay))
    c = scw.Context(0)
    try:
        if path == "tensor":
            c.set_path(scw.SCW_PATH_TENSOR)
        L = scw.Layer.from_numpy(lay, "cuda")
        I = scw.scw_sweep_intensity(c, [L, L], [dev(z), dev(z[:3])], dev(x), dev(y))
        torch.cuda.synchronize()
        assert I[0].dtype == (torch.float32 if dtype == np.complex64 else torch.float64)
        assert np.abs(I[0].cpu().numpy() - ref).max() / ref.max() <= tol
        assert np.abs(I[1].cpu().numpy() - ref[:3]).max() / ref.max() <= tol
    finally:
        c.close()


@pytest.mark.gpu
def test_config4_intensity_full_size_fused(scw):
    """Config 4 (32 wavelengths x 2 layers, one call) on the fused tcgen05 epilogue: every sample of four instances
    against Tier B, all instances against the complex sweep, custom strides, and no complex field written."""
    import torch
    c4 = si.CONFIGS[4]
    x, y, _ = si.grid_coords(c4, 0)
    lays, zs = [], []
    for li in range(len(c4.lams)):
        for l in range(c4.n_layers):
            lays.append(si.make_layer(c4, l, li, dtype=np.complex64))
            zs.append(si.grid_coords(c4, l)[2])
    ctx = scw.Context(0)
    try:
        Ls = [scw.Layer.from_numpy(d, "cuda") for d in lays]
        dz, dx, dy = [dev(z) for z in zs], dev(x), dev(y)
        n0 = ctx.launch_count()
        I = scw.scw_sweep_intensity(ctx, Ls, dz, dx, dy)
        torch.cuda.synchronize()
        assert ctx.launch_count() - n0 == 3                      # twiddles, assembly (weights + images inside), synthesis+detector
        for i in (0, 1, 37, 63):
            ref = oracle.intensity(oracle.tier_b_grid(x=x, y=y, z=zs[i], **lays[i]))
            assert np.abs(I[i].cpu().numpy() - ref).max() / ref.max() <= 4e-4
        # every one of the 64 instances against the plain definition (Tier A): 32 seeded samples each
        for i in range(len(Ls)):
            idx = si.sample_subset(c4, 16 * 256 * 256, 32, lam_index=i // 2, layer=i % 2)
            iz, iy, ix = np.unravel_index(idx, (16, 256, 256))
            Ea = oracle.layer_samples(xyz=np.column_stack([x[ix], y[iy], zs[i][iz]]), **lays[i])
            Ia = (np.abs(Ea) ** 2).sum(axis=1)
            got = I[i][torch.from_numpy(iz).cuda(), torch.from_numpy(iy).cuda(), torch.from_numpy(ix).cuda()].cpu().numpy()
            assert np.abs(got - Ia).max() / float(I[i].max()) <= 4e-4, i
        E = scw.scw_sweep_wavelengths(ctx, Ls, dz, dx, dy)
        torch.cuda.synchronize()
        for i in range(len(Ls)):
            Ie = (E[i].real ** 2 + E[i].imag ** 2).sum(dim=1)
            assert float((I[i] - Ie).abs().max() / Ie.max()) <= 2e-6
        # [Ny][Nx][Fz] output (z fastest) through custom strides
        Fz = len(zs[0])
        out = [torch.zeros((c4.Ny, c4.Nx, Fz), dtype=torch.float32, device="cuda") for _ in Ls[:2]]
        scw.scw_sweep_intensity(ctx, Ls[:2], dz[:2], dx, dy, out=out, strides=(1, c4.Nx * Fz, Fz))
        torch.cuda.synchronize()
        assert float((out[1].permute(2, 0, 1) - I[1]).abs().max()) <= 5e-5 * float(I[1].max())   # other stream-K split
    finally:
        ctx.close()


@pytest.mark.gpu
@pytest.mark.parametrize("U,Vn", [(33, 33), (45, 50)])
def test_intensity_wide_frequency_grids(scw, U, Vn):
    """Fused detector with more than 32 frequencies along u (no 128 spare TMEM columns for the running sum: the other
    accumulation mode of the epilogue), ragged Nx / Ny, custom strides, two instances: against oracle.intensity of
    Tier B and against sum |E|^2 of the complex sweep."""
    import torch
    g = np.random.default_rng(U)
    M, J, R = U * Vn, 96, 3 * U * Vn
    lays = []
    for i in range(2):
        V = ((g.standard_normal((J, R)) + 1j * g.standard_normal((J, R))) / np.sqrt(2 * M)).astype(np.complex64)
        dirs = np.where(np.arange(J) % 2 == 0, 1, -1).astype(np.int8)
        gamma = dirs * (g.uniform(0.2, 1.4, J) + 1j * g.uniform(0.0, 0.2, J))
        c = ((g.standard_normal(J) + 1j * g.standard_normal(J)) / np.sqrt(2)).astype(np.complex64)
        lays.append(dict(U=U, Vn=Vn, X=30.0, Y=28.0, lam=0.9, z_lo=0.0, z_hi=1.3, V=V, c=c, gamma=gamma, dir=dirs))
    Nx, Ny, Fz = 150, 131, 3
    x = np.sort(g.uniform(0, 30, Nx))
    y = np.sort(g.uniform(0, 28, Ny))
    zs = [np.linspace(0.1, 1.2, Fz), np.linspace(0.0, 1.3, Fz)]
    ctx = scw.Context(0)
    try:
        ctx.set_path(scw.SCW_PATH_TENSOR)
        Ls = [scw.Layer.from_numpy(d, "cuda") for d in lays]
        dz, dx, dy = [dev(z) for z in zs], dev(x), dev(y)
        out = [torch.full((Ny, Nx, Fz), float("nan"), dtype=torch.float32, device="cuda") for _ in Ls]   # [y][x][z]
        scw.scw_sweep_intensity(ctx, Ls, dz, dx, dy, out=out, strides=(1, Nx * Fz, Fz))
        E = scw.scw_sweep_wavelengths(ctx, Ls, dz, dx, dy)
        torch.cuda.synchronize()
        for i in range(2):
            I = out[i].permute(2, 0, 1)
            ref = oracle.intensity(oracle.tier_b_grid(x=x, y=y, z=zs[i], **lays[i]))
            assert np.abs(I.cpu().numpy() - ref).max() / ref.max() <= 4e-4
            Ie = (E[i].real ** 2 + E[i].imag ** 2).sum(dim=1)
            assert float((I - Ie).abs().max() / Ie.max()) <= 5e-6
    finally:
        ctx.close()


# ------------------------------------------------------------------------------------------------ window sums, absorbance
def test_window_sum_and_absorbance_closed_forms():
    """Pins for the remaining detector reductions (CPU).  (i) One plane wave: I is flat, so the window sum is the number of
    samples in the window times I.  (ii) Absorbing homogeneous slab, one "+" wave at normal incidence with gamma = n:
    I(z) = I(z_lo) exp(-2 k Im(n) (z - z_lo)), so A = -log10(I(z_hi) / I(z_lo)) = 2 k Im(n) t log10(e) (Beer-Lambert).
    (iii) Band absorbance of equal readings equals the single absorbance; weights act as a weighted mean of S, S0."""
    cfg = si.CONFIGS[0]
    lay = si.make_layer(cfg, dtype=np.complex128)
    M = lay["U"] * lay["Vn"]
    j, m = 6, 40
    V1 = np.zeros_like(lay["V"])
    for comp in range(3):
        V1[j, comp * M + m] = lay["V"][j, comp * M + m]
    one = dict(lay, V=V1)
    x, y, z = np.arange(12) * 0.37, np.arange(9) * 0.51, np.array([0.4, 1.9])
    I = oracle.intensity(oracle.layer_grid(x=x, y=y, z=z, **one))
    S = oracle.window_sum(I, (2, 9, 1, 6))
    assert np.allclose(S, 7 * 5 * I[:, 0, 0], rtol=1e-12)
    assert np.allclose(oracle.window_sum(I), 12 * 9 * I[:, 0, 0], rtol=1e-12)
    # Beer-Lambert slab
    n_slab, lam, t = 1.45 + 0.03j, 0.8, 2.5
    Vs = np.zeros((4, 3), dtype=np.complex128)
    Vs[0, 0] = 1.0                                              # E_x, frequency (0, 0), "+" mode
    slab = dict(U=1, Vn=1, X=3.0, Y=3.0, lam=lam, z_lo=0.0, z_hi=t, V=Vs, c=None,
                gamma=np.array([n_slab, -n_slab, n_slab, -n_slab]), dir=np.array([1, -1, 1, -1], dtype=np.int8))
    slab["c"] = np.array([1.0, 0, 0, 0], dtype=np.complex128)
    Iz = oracle.intensity(oracle.layer_grid(x=np.array([0.3, 1.1]), y=np.array([0.2]), z=np.array([0.0, t]), **slab))
    A = oracle.absorbance(oracle.window_sum(Iz)[1], oracle.window_sum(Iz)[0])
    assert abs(A - 2 * (2 * np.pi / lam) * n_slab.imag * t * np.log10(np.e)) < 1e-12
    assert abs(oracle.band_absorbance([3.0, 3.0], [6.0, 6.0]) - np.log10(2.0)) < 1e-15
    assert abs(oracle.band_absorbance([1.0, 4.0], [2.0, 4.0], w=[1.0, 0.5]) + np.log10(3.0 / 4.0)) < 1e-15


@pytest.mark.gpu
@pytest.mark.parametrize("dtype,tol", [(np.complex64, 4e-4), (np.complex128, 2e-10)])
@pytest.mark.parametrize("want_I", [True, False])
def test_detector_window_sums_and_absorbance(scw, dtype, tol, want_I):
    """scw_sweep_detector: window sums (with and without the per-sample intensity) against oracle.window_sum of Tier A /
    Tier B intensities, ragged grid spanning several output tiles, two instances; then scw_absorbance against the oracle."""
    import torch
    cfg = si.CONFIGS[0]
    lays = [si.make_layer(cfg, dtype=dtype), si.make_layer(cfg, dtype=dtype, lam_index=0, layer=0)]
    lays[1] = dict(lays[1], c=(lays[1]["c"] * 0.5).astype(dtype))
    g = np.random.default_rng(3)
    Nx, Ny, Fz = 150, 140, 3
    x, y = np.sort(g.uniform(0, 8, Nx)), np.sort(g.uniform(0, 8, Ny))
    zs = [np.linspace(0.1, 1.8, Fz), np.linspace(0.0, 2.0, Fz)]
    win = (17, 141, 5, 133)
    ctx = scw.Context(0)
    try:
        Ls = [scw.Layer.from_numpy(d, "cuda") for d in lays]
        I, S = scw.scw_sweep_detector(ctx, Ls, [dev(z) for z in zs], dev(x), dev(y), window=win, want_I=want_I)
        _, S_all = scw.scw_sweep_detector(ctx, Ls, [dev(z) for z in zs], dev(x), dev(y), want_I=False)
        torch.cuda.synchronize()
        assert (I is None) == (not want_I)
        refs = []
        for i in range(2):
            Iref = oracle.intensity(oracle.tier_b_grid(x=x, y=y, z=zs[i], **lays[i]))
            Sref, Sref_all = oracle.window_sum(Iref, win), oracle.window_sum(Iref)
            refs.append(Sref)
            assert np.abs(S[i].cpu().numpy() - Sref).max() / Sref.max() <= tol
            assert np.abs(S_all[i].cpu().numpy() - Sref_all).max() / Sref_all.max() <= tol
            if want_I:
                assert np.abs(I[i].cpu().numpy() - Iref).max() / Iref.max() <= tol
        w = torch.tensor([1.0, 0.5, 2.0], dtype=S[0].dtype, device="cuda")
        A, band = scw.scw_absorbance(ctx, S[1], S[0], w=w, want_band=True)
        torch.cuda.synchronize()
        Aref = oracle.absorbance(refs[1], refs[0])
        assert np.abs(A.cpu().numpy() - Aref).max() <= 10 * tol
        assert abs(float(band) - oracle.band_absorbance(refs[1], refs[0], w=[1.0, 0.5, 2.0])) <= 10 * tol
    finally:
        ctx.close()


@pytest.mark.gpu
def test_detector_errors(scw):
    import torch
    cfg = si.CONFIGS[0]
    lay = si.make_layer(cfg, dtype=np.complex64)
    x, y, z = si.grid_coords(cfg, 0, planes=2, Nx=16, Ny=12)
    ctx = scw.Context(0)
    try:
        L = scw.Layer.from_numpy(lay, "cuda")
        for bad in [(0, 0, 0, 12), (0, 17, 0, 12), (-1, 4, 0, 12), (0, 16, 5, 5), (0, 16, 0, 13)]:
            with pytest.raises(scw.ScwError) as e:
                scw.scw_sweep_detector(ctx, [L], [dev(z)], dev(x), dev(y), window=bad)
            assert e.value.status == 2
        with pytest.raises(scw.ScwError) as e:
            scw.scw_sweep_detector(ctx, [L], [dev(z)], dev(x), dev(y), want_I=False, want_S=False)
        assert e.value.status == 1
        torch.cuda.synchronize()
    finally:
        ctx.close()

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

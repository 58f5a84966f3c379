"""GPU parity at large phases: the range-reduction edge `north_star` singles out ("the phase k(s.r) range-reduced in
fp64 before sincospi").

The complex64 weight and point kernels reduce with the magic constant 1.5*2^20, exact only while |phase| < 2^19
turns; the library keeps every phase inside that window (weights: rint first; points: phases relative to the first
point of the call, reducing loop for blocks beyond the window), so that any finite coordinate gives the oracle's value.
Covered here for complex64 AND complex128, grid and point paths:
  * coordinates shifted by K periods (periodicity, fixes the answer),
  * a thick layer with gamma dz / lambda ~ 1e5 turns,
  * phases just inside and just beyond 2^19 turns.
Tolerances: 2e-4 (complex64).  complex128: 1e-10 + 8 pi 2^-53 max|phase in turns| -- both sides form the phase as a
few fp64 products of magnitude |phase|, each with a rounding error of 2^-53 |phase| turns, before the exact reduction.
"""
import numpy as np
import pytest
import torch

import oracle

pytestmark = pytest.mark.gpu

TWO19 = float(1 << 19)


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


def tol_for(dtype, max_turns):
    return 2e-4 if dtype == np.complex64 else 1e-10 + 8 * np.pi * 2.0 ** -53 * max_turns


def toy_layer(dtype, seed, U=5, Vn=5, lam=0.8, X=4.0, Y=5.0, z_lo=0.0, z_hi=1.5, im_max=0.3, gamma_re=(0.3, 1.4)):
    """M = 25 frequencies, J = 100 modes: large enough for the tcgen05 assembly (2R >= 128, J >= 64)."""
    g = np.random.default_rng(seed)
    M, J, R = U * Vn, 4 * U * Vn, 3 * U * Vn
    V = ((g.standard_normal((J, R)) + 1j * g.standard_normal((J, R))) / np.sqrt(2 * M)).astype(dtype)
    c = ((g.standard_normal(J) + 1j * g.standard_normal(J)) / np.sqrt(2)).astype(dtype)
    dirs = np.where(np.arange(J) % 2 == 0, 1, -1).astype(np.int8)
    gamma = dirs * (g.uniform(*gamma_re, J) + 1j * g.uniform(0.0, im_max, J))
    return dict(U=U, Vn=Vn, X=X, Y=Y, lam=lam, z_lo=z_lo, z_hi=z_hi, V=V, c=c, gamma=gamma, dir=dirs)


# ------------------------------------------------------------------------------------------------ grid path
@pytest.mark.parametrize("dtype,K", [(np.complex64, 10_000), (np.complex128, 100)])
def test_grid_shifted_by_K_periods(scw, ctx, dtype, K):
    """x -> x + K X, y -> y - K Y: every sample against Tier A at the shifted coordinates, and against the unshifted
    field (periodicity; the shifted coordinates carry a representation error of 2^-53 K X)."""
    lay = toy_layer(dtype, seed=1)
    x = np.arange(40) * lay["X"] / 40 + 0.013
    y = np.arange(24) * lay["Y"] / 24 + 0.007
    z = np.linspace(lay["z_lo"], lay["z_hi"], 5)
    xs, ys = x + K * lay["X"], y - K * lay["Y"]
    ref = oracle.layer_grid(x=xs, y=ys, z=z, **lay)
    ref0 = oracle.layer_grid(x=x, y=y, z=z, **lay)
    max_turns = K * (lay["U"] // 2 + lay["Vn"] // 2 + 2)
    tol = tol_for(dtype, max_turns)
    assert rel_err(ref, ref0) <= 1e-10 + 8 * np.pi * 2.0 ** -53 * max_turns          # the oracle itself is periodic
    L = scw.Layer.from_numpy(lay, "cuda")
    E = scw.scw_sweep_wavelengths(ctx, [L], [dev(z)], dev(xs), dev(ys))[0]
    torch.cuda.synchronize()
    assert rel_err(E.cpu().numpy(), ref) <= tol
    assert rel_err(E.cpu().numpy(), ref0) <= tol
    # dense point path (eq. 34 at scattered points) at the same shifted coordinates
    xyz = oracle.grid_points(xs, ys, z)[::7]
    Ep = scw.scw_eval_points(ctx, L, dev(xyz))
    torch.cuda.synchronize()
    refp = oracle.layer_samples(xyz=xyz, **lay)
    assert np.abs(Ep.cpu().numpy() - refp).max() / np.abs(ref).max() <= tol


@pytest.mark.parametrize("path", ["auto", "simt"])
@pytest.mark.parametrize("dtype,thick", [(np.complex64, 1.0e5), (np.complex64, TWO19 - 1.5), (np.complex64, TWO19 + 40.0),
                                         (np.complex64, 3.3e6), (np.complex128, 1.0e4)])
def test_thick_layer_weights(scw, path, dtype, thick):
    """A layer `thick` wavelengths thick with propagating modes (Im gamma = 0 or ~1/thick): gamma dz / lambda reaches
    ~thick turns, incl. just inside / beyond the 2^19-turn window of the magic-constant reduction."""
    c = scw.Context(0)
    try:
        if path == "simt":
            c.set_path(scw.SCW_PATH_SIMT)
        lam = 0.8
        lay = toy_layer(dtype, seed=2, lam=lam, z_lo=0.0, z_hi=thick * lam, im_max=0.0, gamma_re=(0.5, 1.0))
        g = np.random.default_rng(3)
        lay["gamma"] = lay["gamma"] + 1j * lay["dir"] * np.where(np.arange(100) % 3 == 0, g.uniform(0, 2.0 / thick, 100), 0.0)
        lay["gamma"][0] = 1.0                                           # exactly `thick` turns at the far face
        lay["gamma"][1] = -1.0
        x = np.arange(16) * lay["X"] / 16
        y = np.arange(12) * lay["Y"] / 12
        z = np.concatenate([[0.0, thick * lam], g.uniform(0.0, thick * lam, 6)])
        ref = oracle.layer_grid(x=x, y=y, z=z, **lay)
        L = scw.Layer.from_numpy(lay, "cuda")
        E = scw.scw_sweep_wavelengths(c, [L], [dev(z)], dev(x), dev(y))[0]
        torch.cuda.synchronize()
        assert rel_err(E.cpu().numpy(), ref) <= tol_for(dtype, thick)
    finally:
        c.close()


# ------------------------------------------------------------------------------------------------ point path
def planewave_table(dtype, seed, J=300, lam=0.8, im_max=0.05):
    g = np.random.default_rng(seed)
    sx, sy = g.uniform(-0.6, 0.6, J), g.uniform(-0.6, 0.6, J)
    sign = np.where(np.arange(J) % 2 == 0, 1.0, -1.0)
    gamma = sign * (g.uniform(0.4, 1.3, J) + 1j * g.uniform(0.0, im_max, J))
    zref = np.where(sign > 0, 0.0, 1.5)
    p = ((g.standard_normal((J, 3)) + 1j * g.standard_normal((J, 3))) / np.sqrt(2 * J)).astype(dtype)
    return dict(lam=lam, sx=sx, sy=sy, gamma=gamma, zref=zref, p=p)


@pytest.mark.parametrize("dtype,offset", [(np.complex64, 3.2e5), (np.complex64, 4.0e7), (np.complex128, 2.0e3)])
def test_points_far_from_the_origin(scw, ctx, dtype, offset):
    """A compact cloud of points `offset` wavelengths away from the origin in x and y: phases ~ offset turns, far
    beyond 2^19 for the second case; the kernel works relative to the first point of the call."""
    pw = planewave_table(dtype, seed=4)
    g = np.random.default_rng(5)
    n = 1500                                                            # ragged: not a multiple of the block's points
    pts = np.column_stack([offset * pw["lam"] + g.uniform(0, 30, n), -offset * pw["lam"] + g.uniform(0, 30, n),
                           g.uniform(0.0, 1.5, n)])
    ref = oracle.planewaves(xyz=pts, **pw)
    E = scw.scw_eval_points(ctx, scw.PlaneWaves.from_numpy(pw, "cuda"), dev(pts))
    torch.cuda.synchronize()
    assert rel_err(E.cpu().numpy(), ref) <= tol_for(dtype, 2 * 0.6 * offset + 60)


@pytest.mark.parametrize("dtype", [np.complex64, np.complex128])
@pytest.mark.parametrize("extent", [TWO19 - 40.0, TWO19 + 40.0, 6.0e6])
def test_points_cloud_extent_around_the_window(scw, ctx, dtype, extent):
    """Point clouds whose EXTENT reaches the window: one wave with s_x = 1 and Im gamma = 0 puts the relative phase of
    the far points at `extent` turns -- just inside 2^19 (fast loop), just beyond and far beyond (reducing loop); the
    near points of the same call stay on the fast loop (the choice is per block)."""
    pw = planewave_table(dtype, seed=6, im_max=0.0)
    pw["sx"][0], pw["sy"][0], pw["gamma"][0] = 1.0, 0.0, 0.0 + 0.0j
    lam = pw["lam"]
    g = np.random.default_rng(7)
    n_near, n_far = 1100, 900
    near = np.column_stack([g.uniform(0, 20, n_near), g.uniform(0, 20, n_near), g.uniform(0, 1.5, n_near)])
    far = np.column_stack([extent * lam + g.uniform(-3, 0, n_far), g.uniform(0, 20, n_far), g.uniform(0, 1.5, n_far)])
    far[0, 0] = extent * lam                                            # exactly `extent` turns for wave 0
    pts = np.vstack([near[:1] * 0.0, near, far])                        # first point = origin of the relative phases
    ref = oracle.planewaves(xyz=pts, **pw)
    E = scw.scw_eval_points(ctx, scw.PlaneWaves.from_numpy(pw, "cuda"), dev(pts))
    torch.cuda.synchronize()
    tol = tol_for(dtype, extent) if dtype == np.complex64 else 1e-10 + 8 * np.pi * 2.0 ** -53 * extent
    assert rel_err(E.cpu().numpy(), ref) <= tol

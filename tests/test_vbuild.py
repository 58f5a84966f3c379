"""V builder (eq. 33): oracle pins (CPU) and GPU parity through the C ABI.

Pins of oracle.build_V: psi = delta reduces eq. 33 to a Hadamard product; a homogeneous layer built from plane waves with
b = s x p (Faraday) must give back p_z and transversality s.p = 0 (eq. 14) -- only the + sign of reading
c-19 does; the 2-D circular convolution against numpy's FFT (convolution theorem, the paper's own argument at
PAPER.md:366-374) and against a pure-python loop over (u, v) pairs on a 3 x 3 toy.
"""
import math

import numpy as np
import pytest

import oracle
import scw_inputs as si


def random_Q(U, Vn, J, seed, dtype=np.complex128, pad=0):
    g = np.random.default_rng(seed)
    M = U * Vn
    Q = np.zeros((J, 4 * M + pad), dtype=dtype)
    Q[:, :4 * M] = ((g.standard_normal((J, 4 * M)) + 1j * g.standard_normal((J, 4 * M))) / np.sqrt(8 * M)).astype(dtype)
    if pad:
        Q[:, 4 * M:] = 9 + 9j
    psi = ((g.standard_normal(M) + 1j * g.standard_normal(M)) / np.sqrt(2 * M)).astype(dtype)
    psi[M // 2] += 0.5                                            # DC term (1/n^2 average)
    return Q, psi


def test_psi_delta_is_a_hadamard_product():
    U, Vn, lam, X, Y = 5, 3, 0.8, 4.0, 3.0
    M = U * Vn
    Q, _ = random_Q(U, Vn, 11, seed=1)
    psi = np.zeros(M, dtype=np.complex128)
    psi[M // 2] = 0.37 - 0.1j                                     # frequency (0, 0)
    V = oracle.build_V(U=U, Vn=Vn, X=X, Y=Y, lam=lam, Q=Q, psi=psi)
    uu, vv = si.freq_uv(U, Vn)
    sx, sy = lam * uu / X, lam * vv / Y
    assert np.array_equal(V[:, :2 * M], Q[:, :2 * M])
    ref = psi[M // 2] * (sy * Q[:, 2 * M:3 * M] - sx * Q[:, 3 * M:])
    assert np.abs(V[:, 2 * M:] - ref).max() < 1e-15


def test_homogeneous_layer_recovers_pz_and_transversality():
    """Columns of Q = plane waves of a homogeneous medium: p transverse to s = (sx, sy, +-sz), b = s x p.  With
    psi = delta / n^2 the builder must return p_z (so that s.p = 0, eq. 14); the printed minus sign would return -p_z."""
    U, Vn, lam, L, n = 3, 3, 0.8, 3.0, 1.45 + 0.02j
    M = U * Vn
    uu, vv = si.freq_uv(U, Vn)
    Q = np.zeros((4 * M, 4 * M), dtype=np.complex128)
    P = np.zeros((4 * M, 3), dtype=np.complex128)
    S = np.zeros((4 * M, 3), dtype=np.complex128)
    for j in range(4 * M):
        m, pol, d = j // 4, (j // 2) % 2, j % 2
        sx, sy = lam * uu[m] / L, lam * vv[m] / L
        sz = oracle.sz(n, sx, sy) * (1 if d == 0 else -1)
        sb = math.hypot(sx, sy)
        if sb == 0:
            p = np.array([1, 0, 0], dtype=complex) if pol == 0 else np.array([0, 1, 0], dtype=complex)
        elif pol == 0:
            p = np.array([-sy, sx, 0], dtype=complex) / sb
        else:
            p = np.array([sx * sz, sy * sz, -sb * sb], dtype=complex) / (sb * n)
        s = np.array([sx, sy, sz])
        b = np.cross(s, p)                                        # Faraday: b = s x p
        Q[j, m], Q[j, M + m], Q[j, 2 * M + m], Q[j, 3 * M + m] = p[0], p[1], b[0], b[1]
        P[j], S[j] = p, s
    psi = np.zeros(M, dtype=np.complex128)
    psi[M // 2] = 1 / n ** 2
    V = oracle.build_V(U=U, Vn=Vn, X=L, Y=L, lam=lam, Q=Q, psi=psi)
    for j in range(4 * M):
        m = j // 4
        pz = V[j, 2 * M + m]
        assert abs(pz - P[j, 2]) < 1e-14, (j, pz, P[j, 2])
        assert abs(S[j, 0] * V[j, m] + S[j, 1] * V[j, M + m] + S[j, 2] * pz) < 1e-14          # eq. 14
        others = np.delete(V[j, 2 * M:], m)
        assert np.abs(others).max() < 1e-15


@pytest.mark.parametrize("U,Vn", [(3, 3), (5, 4), (4, 6)])
def test_convolution_theorem_and_wrap(U, Vn):
    """Eq. 33 is the 2-D circular convolution of psi with q = s_y b_x - s_x b_y on the (u, v) grid: numpy FFT as the
    independent route (frequency u lives at FFT index u mod U)."""
    lam, X, Y = 0.7, 3.0, 5.0
    M = U * Vn
    Q, psi = random_Q(U, Vn, 6, seed=2)
    alpha = np.arange(1, 7) * (0.5 - 0.25j)
    V = oracle.build_V(U=U, Vn=Vn, X=X, Y=Y, lam=lam, Q=Q, psi=psi, alpha=alpha)
    uu, vv = si.freq_uv(U, Vn)
    sx, sy = lam * uu / X, lam * vv / Y
    q = sy * Q[:, 2 * M:3 * M] - sx * Q[:, 3 * M:]
    def to_fft(a):
        g = np.zeros((Vn, U), dtype=np.complex128)
        g[vv % Vn, uu % U] = a
        return g
    for j in range(Q.shape[0]):
        conv = np.fft.ifft2(np.fft.fft2(to_fft(psi)) * np.fft.fft2(to_fft(q[j])))
        assert np.abs(V[j, 2 * M:] - alpha[j] * conv[vv % Vn, uu % U]).max() < 1e-13
        assert np.abs(V[j, :2 * M] - alpha[j] * Q[j, :2 * M]).max() < 1e-15


def test_bruteforce_pairs_on_3x3():
    U = Vn = 3
    M = 9
    Q, psi = random_Q(U, Vn, 2, seed=3)
    V = oracle.build_V(U=U, Vn=Vn, X=2.0, Y=2.5, lam=0.9, Q=Q, psi=psi)
    wrap = lambda d: (d + 1) % 3 - 1
    for j in range(2):
        for u in (-1, 0, 1):
            for v in (-1, 0, 1):
                acc = 0j
                for up in (-1, 0, 1):
                    for vp in (-1, 0, 1):
                        du, dv = wrap(u - up), wrap(v - vp)
                        md, mp = (dv + 1) * 3 + du + 1, (vp + 1) * 3 + up + 1
                        acc += psi[mp] * (0.9 * dv / 2.5 * Q[j, 2 * M + md] - 0.9 * du / 2.0 * Q[j, 3 * M + md])
                assert abs(V[j, 2 * M + (v + 1) * 3 + u + 1] - acc) < 1e-14


# ------------------------------------------------------------------------------------------------ GPU
def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.gpu
@pytest.mark.parametrize("path", ["auto", "simt"])
@pytest.mark.parametrize("dtype,tol", [(np.complex64, 2e-4), (np.complex128, 1e-10)])
@pytest.mark.parametrize("U,Vn,J,pad,with_alpha", [(3, 3, 36, 0, False), (9, 9, 324, 3, True), (12, 7, 100, 1, True)])
def test_build_V_every_entry(dtype, tol, U, Vn, J, pad, with_alpha, path):
    """scw_build_V against oracle.build_V, every entry: odd / even grids, J != 4M, padded ldQ / ldV, alpha folded or not;
    complex64 on the tcgen05 GEMM where a tile fits (M >= 64), complex128 on DMMA, both on CUDA cores ("simt")."""
    import torch
    import paper_2404_07293_b200 as scw
    M = U * Vn
    Q, psi = random_Q(U, Vn, J, seed=U * 10 + Vn, dtype=dtype, pad=pad)
    g = np.random.default_rng(5)
    alpha = ((g.standard_normal(J) + 1j * g.standard_normal(J)) / np.sqrt(2)).astype(dtype) if with_alpha else None
    lam, X, Y = 0.8, 5.0, 4.0
    ref = oracle.build_V(U=U, Vn=Vn, X=X, Y=Y, lam=lam, Q=Q, psi=psi, alpha=alpha)
    ctx = scw.Context(0)
    try:
        if path == "simt":
            ctx.set_path(scw.SCW_PATH_SIMT)
        out = torch.full((J, 3 * M + pad), 7.0, dtype=dev(Q).dtype, device="cuda")
        V = scw.scw_build_V(ctx, U=U, Vn=Vn, X=X, Y=Y, lam=lam, Q=dev(Q), psi=dev(psi),
                            alpha=None if alpha is None else dev(alpha), out=out)
        torch.cuda.synchronize()
        got = V.cpu().numpy()
        assert np.all(got[:, 3 * M:] == 7.0)                          # padding rows of V untouched
        assert np.abs(got[:, :3 * M] - ref).max() / np.abs(ref).max() <= tol
    finally:
        ctx.close()


@pytest.mark.gpu
def test_build_V_feeds_the_field_evaluation():
    """End to end at config-1 shape (33 x 33, J = 4356, complex64): V from scw_build_V (tcgen05 GEMM) equals the oracle's V on
    sampled columns, and the field evaluated from it equals Tier B evaluated from the oracle's V."""
    import torch
    import paper_2404_07293_b200 as scw
    cfg = si.CONFIGS[1]
    U, Vn, M = cfg.U, cfg.Vn, cfg.U * cfg.Vn
    J = 4 * M
    Q, psi = random_Q(U, Vn, J, seed=77, dtype=np.complex64)
    lay = si.make_layer(cfg, 0, dtype=np.complex64, with_V=False)
    ctx = scw.Context(0)
    try:
        V = scw.scw_build_V(ctx, U=U, Vn=Vn, X=cfg.L, Y=cfg.L, lam=lay["lam"], Q=dev(Q), psi=dev(psi))
        torch.cuda.synchronize()
        cols = np.sort(np.random.default_rng(1).choice(J, 24, replace=False))
        ref = oracle.build_V(U=U, Vn=Vn, X=cfg.L, Y=cfg.L, lam=lay["lam"], Q=Q[cols], psi=psi)
        got = V.cpu().numpy()
        assert np.abs(got[cols] - ref).max() / np.abs(ref).max() <= 2e-4
        # the field from the built V
        x, y, z = si.grid_coords(cfg, 0, planes=2, Nx=64, Ny=48)
        L = scw.Layer(U=U, Vn=Vn, X=cfg.L, Y=cfg.L, lam=lay["lam"], z_lo=lay["z_lo"], z_hi=lay["z_hi"], V=V,
                      gamma=dev(lay["gamma"]), c=dev(lay["c"]), dir=dev(lay["dir"]))
        E = scw.scw_sweep_wavelengths(ctx, [L], [dev(z)], dev(x), dev(y))[0]
        torch.cuda.synchronize()
        Eref = oracle.tier_b_grid(x=x, y=y, z=z, **dict(lay, V=got))
        assert np.abs(E.cpu().numpy() - Eref).max() / np.abs(Eref).max() <= 2e-4
    finally:
        ctx.close()

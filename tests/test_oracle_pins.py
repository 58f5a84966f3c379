"""Pins for the fp64 oracle: what the paper and the mathematics fix (CPU only).

Each test ties one part of oracle/ to something other than itself: hand-derived values
(tests/golden/), closed forms, invariants, library routines (numpy FFT / matmul) that the
oracle does not call on that path, and brute force on tiny inputs.  PAPER.md line numbers
are cited per test.
"""
import cmath
import math
import os

import numpy as np
import pytest

import oracle
import scw_inputs as si


def _read_table(path):
    rows = []
    with open(path) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                rows.append([float(t) for t in line.split()])
    return rows


def _toy_layer(U=3, Vn=3, seed=0, lam=0.9, X=4.0, Y=5.0, z_lo=0.3, z_hi=1.7, dtype=np.complex128,
               ldV=None):
    """Small random layer with complex gamma (both signs), for brute-force checks."""
    g = np.random.default_rng(seed)
    M = U * Vn
    J = 4 * M
    R = 3 * M
    ldV = R if ldV is None else ldV
    V = np.zeros((J, ldV), dtype=dtype)
    V[:, :R] = (g.standard_normal((J, R)) + 1j * g.standard_normal((J, R))).astype(dtype)
    c = (g.standard_normal(J) + 1j * g.standard_normal(J)).astype(dtype)
    dirs = np.where(np.arange(J) % 2 == 0, 1, -1).astype(np.int8)
    gamma = dirs * (g.uniform(0.2, 1.5, J) + 1j * g.uniform(0.0, 0.3, J))
    return dict(U=U, Vn=Vn, X=X, Y=Y, lam=lam, z_lo=z_lo, z_hi=z_hi, V=V, c=c, gamma=gamma,
                dir=dirs)


# --------------------------------------------------------------------------- eq. 6
def test_index_map_golden(golden_dir):
    """hand-derived (u, v) for given m."""
    for U, Vn, m, u, v in _read_table(os.path.join(golden_dir, "index_map.txt")):
        assert oracle.index_map(int(U), int(Vn), int(m)) == (int(u), int(v))


@pytest.mark.parametrize("U,Vn", [(3, 3), (9, 9), (4, 2), (5, 8), (33, 33)])
def test_index_map_bijection_and_forward_formula(U, Vn):
    """m = (v + floor(V/2)) U + u + floor(U/2) inverts the oracle's map; ranges per :79."""
    seen = set()
    for m in range(U * Vn):
        u, v = oracle.index_map(U, Vn, m)
        assert -(U // 2) <= u <= (U - 1) // 2 and -(Vn // 2) <= v <= (Vn - 1) // 2
        assert (v + Vn // 2) * U + u + U // 2 == m
        seen.add((u, v))
    assert len(seen) == U * Vn
    uu, vv = si.freq_uv(U, Vn)         # the input generator uses the same convention
    assert [oracle.index_map(U, Vn, m) for m in range(U * Vn)] == list(zip(uu.tolist(), vv.tolist()))


# --------------------------------------------------------------------------- eq. 2
def test_sz_golden(golden_dir):
    for nr, ni, sx, sy, er, ei in _read_table(os.path.join(golden_dir, "sz_cases.txt")):
        g = oracle.sz(complex(nr, ni), sx, sy)
        assert abs(g - complex(er, ei)) < 1e-15 * max(1.0, abs(complex(er, ei)))


def test_sz_identity_and_branch():
    """gamma^2 + s.s = n^2 and Im gamma >= 0 for random complex n."""
    g = np.random.default_rng(1)
    for _ in range(2000):
        n = complex(g.uniform(0.5, 2.0), g.uniform(0.0, 0.5))
        sx, sy = g.uniform(-2, 2, 2)
        gam = oracle.sz(n, sx, sy)
        assert abs(gam * gam + sx * sx + sy * sy - n * n) < 1e-14 * (abs(n) ** 2 + sx * sx + sy * sy)
        assert gam.imag >= 0 and (gam.imag > 0 or gam.real >= 0)
    # real n, evanescent: exactly on the positive imaginary axis, never -i*sqrt
    assert oracle.sz(1.0, 1.25, 0.0) == complex(0.0, 0.75)
    # the input generator's gamma follows the same rule
    lay = si.make_layer(si.CONFIGS[0], with_V=False)
    assert np.all((lay["dir"] * lay["gamma"]).imag >= 0)


# --------------------------------------------------------------------------- eq. 7
def test_green_closed_forms_and_semigroup():
    """G(A,za,zb) = exp[ik(zb-za)A], k = 2 pi / lambda."""
    assert abs(oracle.green(1.0, 0.0, 0.25, 1.0) - 1j) < 1e-15          # quarter wave -> +i
    assert abs(oracle.green(2.0, 1.0, 1.25, 2.0) - 1j) < 1e-15          # k = 2 pi / lambda
    assert abs(oracle.green(1j, 0.0, 1.0, 2 * math.pi) - math.exp(-1.0)) < 1e-15   # decay for Im A > 0
    assert oracle.green(0.7 + 0.2j, 0.4, 0.4, 1.3) == 1.0
    g = np.random.default_rng(2)
    for _ in range(200):
        A = complex(g.uniform(-2, 2), g.uniform(-0.3, 0.3))
        a, b, c = g.uniform(-1, 1, 3)
        lam = g.uniform(0.5, 1.5)
        lhs = oracle.green(A, a, b, lam) * oracle.green(A, b, c, lam)
        rhs = oracle.green(A, a, c, lam)
        assert abs(lhs - rhs) < 1e-13 * max(1.0, abs(rhs))
        ref = cmath.exp(1j * (2 * math.pi / lam) * (b - a) * A)          # eq. 7 retyped, large-phase safe here
        assert abs(oracle.green(A, a, b, lam) - ref) < 1e-13 * abs(ref)


def test_reference_plane_invariant():
    """|w_j / c_j| <= 1 inside the layer, = 1 on the mode's own face (reading c-1);
    referencing the wrong face breaks it."""
    lay = si.make_layer(si.CONFIGS[0], with_V=False)
    z = np.linspace(lay["z_lo"], lay["z_hi"], 33)
    W = oracle.tier_b_weights(z=z, **lay)
    ratio = np.abs(W) / np.abs(lay["c"])[:, None]
    assert ratio.max() <= 1.0 + 1e-14
    plus = lay["dir"] > 0
    assert np.allclose(ratio[plus, 0], 1.0, atol=1e-14) and np.allclose(ratio[~plus, -1], 1.0, atol=1e-14)
    wrong = dict(lay, dir=(-lay["dir"]).astype(np.int8))
    ratio_wrong = np.abs(oracle.tier_b_weights(z=z, **wrong)) / np.abs(lay["c"])[:, None]
    assert ratio_wrong.max() > 1.0 + 1e-3
    # dir=None derives the face from the sign of gamma
    auto = dict(lay, dir=None)
    assert np.array_equal(oracle.tier_b_weights(z=z, **auto), W)


def test_reference_face_derived_from_gamma_in_tier_a(golden_dir):
    """dir = NULL in Tier A (the C branch scwo_dir): the face of every mode against the hand-derived table
    tests/golden/dir_cases.txt (readings c-1, c-3), through the single-mode closed form
    E = c V exp(i 2 pi (u x/X + v y/Y)) exp(i k gamma (z - zref)); then dir = None must equal the explicit dir on the
    whole toy, and |E| / |c V| <= 1 inside the layer with the derived faces (= 1 on the mode's own face)."""
    rows = _read_table(os.path.join(golden_dir, "dir_cases.txt"))
    J = len(rows)
    U = Vn = 3
    M = 9
    g = np.random.default_rng(21)
    z_lo, z_hi, lam, X, Y = 0.3, 1.7, 0.9, 4.0, 5.0
    gamma = np.array([complex(r[0], r[1]) for r in rows])
    face = np.array([int(r[2]) for r in rows])
    V = (g.standard_normal((J, 3 * M)) + 1j * g.standard_normal((J, 3 * M)))
    c = g.standard_normal(J) + 1j * g.standard_normal(J)
    base = dict(U=U, Vn=Vn, X=X, Y=Y, lam=lam, z_lo=z_lo, z_hi=z_hi, gamma=gamma)
    k = 2 * math.pi / lam
    xyz = np.column_stack([g.uniform(0, 4, 9), g.uniform(0, 5, 9), np.linspace(z_lo, z_hi, 9)])
    for j in range(J):                      # one mode, one frequency at a time: closed form with the table's face
        m, comp = j % M, j % 3
        V1 = np.zeros_like(V)
        V1[j, comp * M + m] = V[j, comp * M + m]
        E = oracle.layer_samples(xyz=xyz, V=V1, c=c, dir=None, **base)
        u, v = m % 3 - 1, m // 3 - 1
        zref = z_lo if face[j] == 0 else z_hi
        for s, (x, y, z) in enumerate(xyz):
            ref = (c[j] * V1[j, comp * M + m] * cmath.exp(2j * math.pi * (u * x / X + v * y / Y))
                   * cmath.exp(1j * k * gamma[j] * (z - zref)))
            assert abs(E[s, comp] - ref) < 1e-13 * abs(ref), (j, gamma[j])
        ratio = np.abs(E[:, comp]) / abs(c[j] * V1[j, comp * M + m])
        assert ratio.max() <= 1.0 + 1e-13                       # decays inside the layer (eq. 30)
        own = 0 if face[j] == 0 else -1                          # xyz[0] is on z_lo, xyz[-1] on z_hi
        assert abs(ratio[own] - 1.0) < 1e-13
    dirs = np.where(face == 0, 1, -1).astype(np.int8)
    E_auto = oracle.layer_samples(xyz=xyz, V=V, c=c, dir=None, **base)
    E_expl = oracle.layer_samples(xyz=xyz, V=V, c=c, dir=dirs, **base)
    assert np.array_equal(E_auto, E_expl)
    E_flip = oracle.layer_samples(xyz=xyz, V=V, c=c, dir=(-dirs).astype(np.int8), **base)
    assert np.abs(E_flip - E_expl).max() > 1e-3 * np.abs(E_expl).max()       # the faces matter
    # Tier B's python mirror takes the same decisions
    W_auto = oracle.tier_b_weights(z=xyz[:, 2], c=c, dir=None, **base)
    W_expl = oracle.tier_b_weights(z=xyz[:, 2], c=c, dir=dirs, **base)
    assert np.array_equal(W_auto, W_expl)


# --------------------------------------------------------------------------- Tier A closed forms
@pytest.mark.parametrize("j,m,comp", [(0, 0, 0), (5, 7, 1), (22, 4, 2), (35, 8, 2)])
def test_single_mode_single_frequency_closed_form(j, m, comp):
    """One nonzero V entry: E = c V exp(i 2 pi (u x/X + v y/Y)) exp(i k gamma dz) (eq. 10 + eq. 30)."""
    lay = _toy_layer(seed=3)
    M = 9
    V = np.zeros_like(lay["V"])
    V[j, comp * M + m] = lay["V"][j, comp * M + m]
    lay["V"] = V
    g = np.random.default_rng(4)
    xyz = np.column_stack([g.uniform(-3, 9, 20), g.uniform(-3, 9, 20), g.uniform(0.3, 1.7, 20)])
    E = oracle.layer_samples(xyz=xyz, **lay)
    u, v = m % 3 - 1, m // 3 - 1
    k = 2 * math.pi / lay["lam"]
    for s, (x, y, z) in enumerate(xyz):
        zref = lay["z_lo"] if lay["dir"][j] > 0 else lay["z_hi"]
        ref = (lay["c"][j] * V[j, comp * M + m]
               * cmath.exp(2j * math.pi * (u * x / lay["X"] + v * y / lay["Y"]))
               * cmath.exp(1j * k * lay["gamma"][j] * (z - zref)))
        exp_abs = abs(lay["c"][j] * V[j, comp * M + m]) * math.exp(-k * lay["gamma"][j].imag * (z - zref))
        assert abs(E[s, comp] - ref) < 1e-13 * abs(ref)
        assert abs(abs(E[s, comp]) - exp_abs) < 1e-13 * exp_abs
        others = [cc for cc in range(3) if cc != comp]
        assert np.all(E[s, others] == 0)


def _spectrum_at_lower_face(lay):
    """At z = z_lo with only '+' modes non-zero every propagator is 1, so P = V c (library matmul)."""
    c = np.where(lay["dir"] > 0, lay["c"], 0)
    R = 3 * lay["U"] * lay["Vn"]
    return dict(lay, c=c), lay["V"][:, :R].T @ c


@pytest.mark.parametrize("U,Vn,Nx,Ny", [(3, 3, 3, 3), (3, 3, 8, 6), (5, 3, 8, 4)])
def test_grid_equals_scaled_ifft2(U, Vn, Nx, Ny):
    """eq. 10 on a commensurate grid is an inverse DFT: E_comp = Nx Ny ifft2(S),
    S[v mod Ny, u mod Nx] = P_comp[u, v] (numpy FFT; not used by the oracle)."""
    lay = _toy_layer(U=U, Vn=Vn, seed=5)
    lay, P = _spectrum_at_lower_face(lay)
    M = U * Vn
    x = np.arange(Nx) * lay["X"] / Nx
    y = np.arange(Ny) * lay["Y"] / Ny
    E = oracle.layer_grid(x=x, y=y, z=np.array([lay["z_lo"]]), **lay)[0]
    uu, vv = si.freq_uv(U, Vn)
    for comp in range(3):
        S = np.zeros((Ny, Nx), dtype=np.complex128)
        np.add.at(S, (vv % Ny, uu % Nx), P[comp * M:(comp + 1) * M])
        ref = Nx * Ny * np.fft.ifft2(S)
        assert np.abs(E[comp] - ref).max() < 1e-12 * np.abs(ref).max()


def test_parseval():
    """sum_xy |E_comp|^2 = Nx Ny sum_m |P_comp,m|^2 when Nx >= U, Ny >= V over one period."""
    lay = _toy_layer(U=3, Vn=5, seed=6)
    lay, P = _spectrum_at_lower_face(lay)
    M, Nx, Ny = 15, 4, 7
    x = np.arange(Nx) * lay["X"] / Nx
    y = np.arange(Ny) * lay["Y"] / Ny
    E = oracle.layer_grid(x=x, y=y, z=np.array([lay["z_lo"]]), **lay)[0]
    for comp in range(3):
        lhs = (np.abs(E[comp]) ** 2).sum()
        rhs = Nx * Ny * (np.abs(P[comp * M:(comp + 1) * M]) ** 2).sum()
        assert abs(lhs - rhs) < 1e-12 * rhs


def test_periodicity_and_real_field():
    """E(x+X, y, z) = E(x, y+Y, z) = E(x,y,z); Hermitian spectrum => real field."""
    lay = _toy_layer(seed=7)
    g = np.random.default_rng(8)
    xyz = np.column_stack([g.uniform(0, 4, 12), g.uniform(0, 5, 12), g.uniform(0.3, 1.7, 12)])
    E0 = oracle.layer_samples(xyz=xyz, **lay)
    for shift in ([lay["X"], 0, 0], [0, lay["Y"], 0], [-2 * lay["X"], 3 * lay["Y"], 0]):
        E1 = oracle.layer_samples(xyz=xyz + np.array(shift), **lay)
        assert np.abs(E1 - E0).max() < 1e-12 * np.abs(E0).max()
    # Hermitian: one '+' mode evaluated on its own face (w = 1), V[(comp,-u,-v)] = conj V[(comp,u,v)]
    M = 9
    col = g.standard_normal(3 * M) + 1j * g.standard_normal(3 * M)
    for comp in range(3):
        blk = col[comp * M:(comp + 1) * M]
        col[comp * M:(comp + 1) * M] = 0.5 * (blk + np.conj(blk[::-1]))   # m -> M-1-m flips (u,v)
    V = np.zeros_like(lay["V"])
    V[0, :3 * M] = col
    herm = dict(lay, V=V, c=None)
    xyz[:, 2] = lay["z_lo"]
    E = oracle.layer_samples(xyz=xyz, **herm)
    assert np.abs(E.imag).max() < 1e-13 * np.abs(E.real).max()


# --------------------------------------------------------------------------- homogeneous layer
def _homogeneous_layer(U=3, Vn=3, n=1.45 + 0.02j, lam=0.8, L=3.0, z_lo=0.0, z_hi=1.2, seed=9):
    """Each column of V is one TE or TM plane wave of a homogeneous medium (SURVEY 8(c) pins)."""
    g = np.random.default_rng(seed)
    M = U * Vn
    J = 4 * M
    uu, vv = si.freq_uv(U, Vn)
    V = np.zeros((J, 3 * M), dtype=np.complex128)
    gamma = np.zeros(J, dtype=np.complex128)
    dirs = np.zeros(J, dtype=np.int8)
    waves = []
    for j in range(J):
        m, pol, d = j // 4, (j // 2) % 2, j % 2
        sx, sy = lam * uu[m] / L, lam * vv[m] / L
        szp = oracle.sz(n, sx, sy)
        s_z = szp if d == 0 else -szp
        sb = math.hypot(sx, sy)
        if sb == 0:
            p = np.array([1, 0, 0], dtype=complex) if pol == 0 else np.array([0, 1, 0], dtype=complex)
        elif pol == 0:                                   # TE
            p = np.array([-sy, sx, 0], dtype=complex) / sb
        else:                                            # TM, transverse to (sx, sy, s_z)
            p = np.array([sx * s_z, sy * s_z, -sb * sb], dtype=complex) / (sb * n)
        assert abs(sx * p[0] + sy * p[1] + s_z * p[2]) < 1e-14          # eq. 14: s.p = 0
        for comp in range(3):
            V[j, comp * M + m] = p[comp]
        gamma[j] = s_z
        dirs[j] = 1 if d == 0 else -1
        waves.append((sx, sy, s_z, p))
    c = g.standard_normal(J) + 1j * g.standard_normal(J)
    lay = dict(U=U, Vn=Vn, X=L, Y=L, lam=lam, z_lo=z_lo, z_hi=z_hi, V=V, c=c, gamma=gamma, dir=dirs)
    return lay, waves


def test_homogeneous_layer_plane_waves():
    """Dense Tier A, the plane-wave form and the analytic sum of eq. 9-10 agree; div E = 0 (eq. 13-14)."""
    lay, waves = _homogeneous_layer()
    g = np.random.default_rng(10)
    xyz = np.column_stack([g.uniform(0, 3, 10), g.uniform(0, 3, 10), g.uniform(0.0, 1.2, 10)])
    E_dense = oracle.layer_samples(xyz=xyz, **lay)
    k = 2 * math.pi / lay["lam"]
    ref = np.zeros((10, 3), dtype=complex)
    for s, (x, y, z) in enumerate(xyz):
        for j, (sx, sy, s_z, p) in enumerate(waves):
            zref = lay["z_lo"] if lay["dir"][j] > 0 else lay["z_hi"]
            ref[s] += lay["c"][j] * p * cmath.exp(1j * k * (sx * x + sy * y + s_z * (z - zref)))
    assert np.abs(E_dense - ref).max() < 1e-12 * np.abs(ref).max()
    modes = dict(lam=lay["lam"], sx=np.array([w[0] for w in waves]), sy=np.array([w[1] for w in waves]),
                 gamma=lay["gamma"], zref=np.where(lay["dir"] > 0, lay["z_lo"], lay["z_hi"]),
                 p=np.ascontiguousarray(np.array([w[3] for w in waves]) * lay["c"][:, None]))
    E_pw = oracle.planewaves(xyz=xyz, **modes)
    assert np.abs(E_pw - ref).max() < 1e-12 * np.abs(ref).max()
    # divergence by central differences of the oracle itself
    h = 1e-4
    div = np.zeros(10, dtype=complex)
    for ax in range(3):
        d = np.zeros(3)
        d[ax] = h
        div += (oracle.layer_samples(xyz=xyz + d, **lay)[:, ax]
                - oracle.layer_samples(xyz=xyz - d, **lay)[:, ax]) / (2 * h)
    assert np.abs(div).max() < 1e-5 * k * np.abs(ref).max()


# --------------------------------------------------------------------------- brute force / identities
def test_bruteforce_eq3_on_3x3_toy():
    """Discrete eq. 3 in (k, s) form, E = sum p exp[ik s.(r - r_ref)], pure python on a 3x3 toy."""
    lay = _toy_layer(seed=11)
    M, J = 9, 36
    k = 2 * math.pi / lay["lam"]
    g = np.random.default_rng(12)
    xyz = np.column_stack([g.uniform(0, 4, 5), g.uniform(0, 5, 5), g.uniform(-0.5, 2.5, 5)])  # z also outside
    E = oracle.layer_samples(xyz=xyz, **lay)
    for s, (x, y, z) in enumerate(xyz):
        ref = [0j, 0j, 0j]
        for j in range(J):
            zref = lay["z_lo"] if j % 2 == 0 else lay["z_hi"]
            for m in range(M):
                u, v = m % 3 - 1, m // 3 - 1
                sx = lay["lam"] * u / lay["X"]            # eq. 6: s = (2 pi / k)(u/X, v/Y)
                sy = lay["lam"] * v / lay["Y"]
                ph = cmath.exp(1j * k * (sx * x + sy * y + lay["gamma"][j] * (z - zref)))
                for comp in range(3):
                    ref[comp] += lay["c"][j] * lay["V"][j, comp * M + m] * ph
        assert np.abs(E[s] - np.array(ref)).max() < 1e-12 * np.abs(np.array(ref)).max()


def test_diag_alpha_identity_linearity_and_ld():
    """Q G alpha = Q diag(alpha) g; linear in c; ldV padding and complex64 V are honoured."""
    lay = _toy_layer(seed=13)
    g = np.random.default_rng(14)
    xyz = np.column_stack([g.uniform(0, 4, 6), g.uniform(0, 5, 6), g.uniform(0.3, 1.7, 6)])
    E = oracle.layer_samples(xyz=xyz, **lay)
    folded = dict(lay, V=np.ascontiguousarray(lay["V"] * lay["c"][:, None]), c=None)
    assert np.abs(oracle.layer_samples(xyz=xyz, **folded) - E).max() < 1e-13 * np.abs(E).max()
    c2 = g.standard_normal(36) + 1j * g.standard_normal(36)
    E2 = oracle.layer_samples(xyz=xyz, **dict(lay, c=c2))
    E12 = oracle.layer_samples(xyz=xyz, **dict(lay, c=lay["c"] + 2 * c2))
    assert np.abs(E12 - (E + 2 * E2)).max() < 1e-12 * np.abs(E12).max()
    padded = np.full((36, 31), 7.0 + 7.0j)
    padded[:, :27] = lay["V"]
    assert np.array_equal(oracle.layer_samples(xyz=xyz, **dict(lay, V=padded)), E)
    lay32 = dict(lay, V=lay["V"].astype(np.complex64))
    E32 = oracle.layer_samples(xyz=xyz, **lay32)
    E32ref = oracle.layer_samples(xyz=xyz, **dict(lay, V=lay32["V"].astype(np.complex128)))
    assert np.array_equal(E32, E32ref)


def test_tier_b_matches_tier_a():
    """The factored reference against the plain definition."""
    cfg = si.CONFIGS[0]
    lay = si.make_layer(cfg)
    x, y, z = si.grid_coords(cfg, 0, planes=3, Nx=5, Ny=4)
    Ea = oracle.layer_grid(x=x, y=y, z=z, **lay)
    Eb = oracle.tier_b_grid(x=x, y=y, z=z, **lay)
    assert Ea.shape == Eb.shape == (3, 3, 4, 5)
    assert np.abs(Ea - Eb).max() < 1e-12 * np.abs(Ea).max()
    xyz = si.make_points(cfg, n=16)
    Ep = oracle.tier_b_points(xyz=xyz, **lay)
    assert np.abs(Ep - oracle.layer_samples(xyz=xyz, **lay)).max() < 1e-12 * np.abs(Ep).max()
    # the spectrum on the lower face with '+' modes only is a plain V c
    lay_p, P = _spectrum_at_lower_face(lay)
    Pb = oracle.tier_b_spectra(z=np.array([lay["z_lo"]]), **lay_p)[:, 0]
    assert np.abs(Pb - P).max() < 1e-13 * np.abs(P).max()


def test_input_recipe_shapes_and_determinism():
    cfg = si.CONFIGS[0]
    a, b = si.make_layer(cfg), si.make_layer(cfg)
    assert a["V"].shape == (324, 243) and a["V"].dtype == np.complex128
    assert np.array_equal(a["V"], b["V"]) and np.array_equal(a["gamma"], b["gamma"])
    assert abs((np.abs(a["V"]) ** 2).mean() * 81 - 1.0) < 0.05      # entries ~ CN(0, 1/M)
    assert np.array_equal(a["dir"][:4], [1, -1, 1, -1])
    c4 = si.CONFIGS[4]
    assert len(c4.lams) == 32 and c4.lams[0] == 0.5 and c4.lams[-1] == 1.5
    zi = si.stack_interfaces(si.CONFIGS[1])
    assert len(zi) == 5 and np.all(np.diff(zi) >= 1.0) and np.all(np.diff(zi) <= 3.0)
    pw = si.make_planewaves(si.CONFIGS[3])
    assert pw["p"].shape == (4356, 3) and pw["p"].dtype == np.complex64
    lay2 = si.make_layer(si.CONFIGS[2], with_V=False)
    assert (np.abs(lay2["gamma"].imag) > 0.5).mean() > 0.15          # evanescent subset present

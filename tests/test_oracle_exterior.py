"""CPU pins of the exterior-field oracle (eq. 9-10).

The oracle's eq. 9 is checked against closed forms typed here, against the textbook Fresnel problem (continuity of
the tangential field AND of its z-derivative across a bare interface -- fails if the reflected wave carried +s_z),
against the decay of evanescent orders away from their interface, and against the pinned plane-wave oracle.
"""
import numpy as np

import oracle
import scw_inputs as si

ABOVE, BELOW = oracle.SIDE_ABOVE, oracle.SIDE_BELOW


def one_freq(U, Vn, m, vec, dtype=np.complex128):
    p = np.zeros((U * Vn, 3), dtype=dtype)
    p[m] = vec
    return p


def test_single_incident_wave_closed_form():
    """One incident order, no reflection: E = p exp(i 2 pi (u x/X + v y/Y)) exp(i k s_z (z - z_inc)), s_z typed here."""
    U, Vn, X, Y, lam, n = 5, 3, 4.0, 6.0, 0.5, 1.5
    for m, (u, v) in ((7, (0, 0)), (13, (1, 1)), (1, (-1, -1))):            # m = (v + 1) * 5 + (u + 2)
        assert oracle.index_map(U, Vn, m) == (u, v)
        vec = np.array([0.3 - 0.1j, -0.7j, 0.2])
        xyz = np.array([[0.3, 1.1, -0.9], [3.7, 5.5, -0.2], [1.0, 2.0, -2.5]])
        E = oracle.exterior_samples(side=ABOVE, U=U, Vn=Vn, X=X, Y=Y, lam=lam, n=n, z_face=0.0, z_inc=-1.0,
                                    p_face=np.zeros((U * Vn, 3), complex), p_inc=one_freq(U, Vn, m, vec), xyz=xyz)
        sx, sy = lam * u / X, lam * v / Y
        s_z = np.sqrt(n * n - sx * sx - sy * sy)                             # real, propagating
        ref = vec[None, :] * np.exp(2j * np.pi * (u * xyz[:, 0] / X + v * xyz[:, 1] / Y)
                                    + 2j * np.pi / lam * s_z * (xyz[:, 2] + 1.0))[:, None]
        assert np.abs(E - ref).max() <= 1e-13


def fresnel_te(n1, n2, sx):
    kz1, kz2 = np.sqrt(n1 * n1 - sx * sx + 0j), np.sqrt(n2 * n2 - sx * sx + 0j)
    return (kz1 - kz2) / (kz1 + kz2), 2 * kz1 / (kz1 + kz2)


def test_fresnel_interface_continuity():
    """Bare interface (z_0 = z_L = 0) between n = 1 and n = 1.5 + 0.1i, TE wave (E along y): with the textbook Fresnel
    r, t as reflected / transmitted amplitudes, E_y and dE_y/dz are continuous at z = 0 (Maxwell)."""
    U, Vn, X, Y, lam = 9, 1, 8.0, 8.0, 1.0
    n1, n2 = 1.0, 1.5 + 0.1j
    for u in (0, 2, 4):
        m = u + 4
        sx = lam * u / X
        r, t = fresnel_te(n1, n2, sx)
        yhat = np.array([0.0, 1.0, 0.0])
        above = dict(side=ABOVE, U=U, Vn=Vn, X=X, Y=Y, lam=lam, n=n1, z_face=0.0, z_inc=0.0,
                     p_face=one_freq(U, Vn, m, r * yhat), p_inc=one_freq(U, Vn, m, yhat))
        below = dict(side=BELOW, U=U, Vn=Vn, X=X, Y=Y, lam=lam, n=n2, z_face=0.0, p_face=one_freq(U, Vn, m, t * yhat))
        h = 1e-4
        pts = lambda zs: np.array([[0.37, 0.0, z] for z in zs])
        Ea = oracle.exterior_samples(xyz=pts([0.0, -h, -2 * h]), **above)[:, 1]
        Eb = oracle.exterior_samples(xyz=pts([0.0, h, 2 * h]), **below)[:, 1]
        assert abs(Ea[0] - Eb[0]) <= 1e-13                                    # 1 + r = t
        da = -(-3 * Ea[0] + 4 * Ea[1] - Ea[2]) / (2 * h)                      # one-sided second-order differences
        db = (-3 * Eb[0] + 4 * Eb[1] - Eb[2]) / (2 * h)
        assert abs(da - db) <= 1e-4 * abs(db)
        # the wrong sign for the reflected wave breaks the derivative match at order one
        wrong = (1j * 2 * np.pi / lam) * np.sqrt(n1 * n1 - sx * sx) * (1 + r) * np.exp(2j * np.pi * u * 0.37 / X)
        assert abs(wrong - db) > 1e-2 * abs(db) or abs(r) < 1e-3


def test_evanescent_orders_decay_away_from_their_interface():
    U, Vn, X, Y, lam = 9, 9, 2.0, 2.0, 1.0                                   # |s| up to 2.8 > n: evanescent orders
    m = 80                                                                   # (u, v) = (4, 4): |s| = 2.83
    vec = np.array([1.0, 0.5j, -0.3])
    zs = np.array([0.0, 0.1, 0.2, 0.4])
    up = oracle.exterior_samples(side=ABOVE, U=U, Vn=Vn, X=X, Y=Y, lam=lam, n=1.0, z_face=0.0,
                                 p_face=one_freq(U, Vn, m, vec), xyz=np.stack([0 * zs, 0 * zs, -zs], 1))
    dn = oracle.exterior_samples(side=BELOW, U=U, Vn=Vn, X=X, Y=Y, lam=lam, n=1.5, z_face=3.0,
                                 p_face=one_freq(U, Vn, m, vec), xyz=np.stack([0 * zs, 0 * zs, 3.0 + zs], 1))
    for E, n in ((up, 1.0), (dn, 1.5)):
        a = np.abs(E[:, 0])
        assert np.all(np.diff(a) < 0) and abs(a[0] - 1.0) <= 1e-14
        kappa = 2 * np.pi / lam * np.sqrt(8.0 - n * n)                        # |s|^2 = 8
        assert np.allclose(a, np.exp(-kappa * zs), rtol=1e-12)


def test_exterior_equals_pinned_planewave_oracle_and_is_periodic():
    """The eq. 9-10 oracle against the (separately pinned) plane-wave Tier A with the wave list written out here."""
    cfg = si.CONFIGS[0]
    for side in (ABOVE, BELOW):
        ext = si.make_exterior(cfg, side, dtype=np.complex128)
        U, Vn, M, lam = ext["U"], ext["Vn"], ext["U"] * ext["Vn"], ext["lam"]
        g = np.random.default_rng(3)
        xyz = g.uniform(0, 8, (40, 3))
        xyz[:, 2] = -xyz[:, 2] if side == ABOVE else ext["z_face"] + xyz[:, 2]
        E = oracle.exterior_samples(xyz=xyz, **ext)
        u, v = si.freq_uv(U, Vn)
        sx, sy = lam * u / ext["X"], lam * v / ext["Y"]
        s_z = np.array([oracle.sz(ext["n"], a, b) for a, b in zip(sx, sy)])
        if side == ABOVE:
            pw = dict(lam=lam, sx=np.tile(sx, 2), sy=np.tile(sy, 2), gamma=np.concatenate([-s_z, s_z]),
                      zref=np.concatenate([np.full(M, ext["z_face"]), np.full(M, ext["z_inc"])]),
                      p=np.ascontiguousarray(np.concatenate([ext["p_face"], ext["p_inc"]])))
        else:
            pw = dict(lam=lam, sx=sx, sy=sy, gamma=s_z, zref=np.full(M, ext["z_face"]), p=ext["p_face"])
        ref = oracle.planewaves(xyz=xyz, **pw)
        assert np.abs(E - ref).max() <= 1e-12 * np.abs(ref).max()
        shifted = xyz + np.array([ext["X"], -2 * ext["Y"], 0.0])
        assert np.abs(oracle.exterior_samples(xyz=shifted, **ext) - E).max() <= 1e-11 * np.abs(E).max()

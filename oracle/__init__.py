"""fp64 CPU oracle for the sCWatter field-evaluation hot path -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
leg may import this package.  It never imports the CUDA package and shares no code
with it.  Citations are PAPER.md line numbers (arxiv 2404.07293).

Tier A  (scw_oracle.c)  : the plain definition -- eq. 34 with eq. 10's factor, one
                          term at a time (sample, mode j, frequency m), long-double sums.
Tier B  (tier_b_* here) : the paper's own factored algorithm O(M^2 Fz + M F)
                           in numpy complex128, a separate
                          statement used to compare *every* sample of the large
                          configs; it is itself validated against Tier A in
                          tests/test_oracle_pins.py.

A "layer" is passed as keyword data (numpy arrays, python scalars):
  U, Vn, X, Y, lam, z_lo, z_hi, V (shape (J, ldV): column-major [ldV x J], complex64 or
  complex128), c ((J,) complex or None), gamma ((J,) complex128), dir ((J,) int8 or None).
"""
import ctypes
import os

import numpy as np

from .build import build as _build

_LIB = None


def lib():
    global _LIB
    if _LIB is None:
        path = _build()
        L = ctypes.CDLL(path)
        dp = ctypes.c_void_p
        L.scwo_threads.restype = ctypes.c_int
        L.scwo_set_threads.argtypes = [ctypes.c_int]
        L.scwo_sz.argtypes = [ctypes.c_double] * 4 + [dp]
        L.scwo_index_map.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp]
        L.scwo_green.argtypes = [ctypes.c_double] * 5 + [dp]
        L.scwo_layer_samples.argtypes = [
            ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_double,
            ctypes.c_double, ctypes.c_double, ctypes.c_int64,
            dp, ctypes.c_int, ctypes.c_int64, dp, dp, dp, ctypes.c_int64, dp, dp]
        L.scwo_planewaves.argtypes = [
            ctypes.c_int64, ctypes.c_double, dp, dp, dp, dp, dp, ctypes.c_int,
            ctypes.c_int64, dp, dp]
        _LIB = L
    return _LIB


def threads() -> int:
    return int(lib().scwo_threads())


def set_threads(n: int) -> None:
    lib().scwo_set_threads(int(n))


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


# ----------------------------------------------------------------------------- small pieces
def sz(n, sx, sy) -> complex:
    """eq. 2, branch Im >= 0."""
    out = np.zeros(2)
    n = complex(n)
    lib().scwo_sz(n.real, n.imag, float(sx), float(sy), _ptr(out))
    return complex(out[0], out[1])


def index_map(U: int, Vn: int, m: int):
    """eq. 6 index map: m -> (u, v)."""
    u = ctypes.c_int()
    v = ctypes.c_int()
    lib().scwo_index_map(U, Vn, m, ctypes.byref(u), ctypes.byref(v))
    return u.value, v.value


def green(A, za, zb, lam) -> complex:
    """eq. 7: G(A, z_a, z_b) = exp[ik (z_b - z_a) A]."""
    out = np.zeros(2)
    A = complex(A)
    lib().scwo_green(A.real, A.imag, float(za), float(zb), float(lam), _ptr(out))
    return complex(out[0], out[1])


# ----------------------------------------------------------------------------- Tier A
def _prep_layer(V, c, gamma, dir):
    assert V.ndim == 2 and V.flags.c_contiguous and V.dtype in (np.complex64, np.complex128)
    J, ldV = V.shape
    gamma = np.ascontiguousarray(gamma, dtype=np.complex128)
    assert gamma.shape == (J,)
    c128 = None if c is None else np.ascontiguousarray(c, dtype=np.complex128)
    d8 = None if dir is None else np.ascontiguousarray(dir, dtype=np.int8)
    return J, ldV, gamma, c128, d8


def layer_samples(*, U, Vn, X, Y, lam, z_lo, z_hi, V, gamma, c=None, dir=None, xyz, **_):
    """Tier A at arbitrary samples xyz [n,3] -> E [n,3] complex128."""
    J, ldV, gamma, c128, d8 = _prep_layer(V, c, gamma, dir)
    assert ldV >= 3 * U * Vn
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    n = xyz.shape[0]
    E = np.zeros((n, 3), dtype=np.complex128)
    lib().scwo_layer_samples(U, Vn, X, Y, lam, z_lo, z_hi, J, _ptr(V),
                             int(V.dtype == np.complex64), ldV, _ptr(c128), _ptr(gamma),
                             _ptr(d8), n, _ptr(xyz), _ptr(E))
    return E


def grid_points(x, y, z):
    """xyz [Fz*Ny*Nx, 3] in the planar output order [z][y][x] (x fastest)."""
    zz, yy, xx = np.meshgrid(z, y, x, indexing="ij")
    return np.stack([xx.ravel(), yy.ravel(), zz.ravel()], axis=1)


def layer_grid(*, x, y, z, **layer):
    """Tier A on a rectilinear grid -> E [Fz, 3, Ny, Nx] complex128 (planar layout)."""
    E = layer_samples(xyz=grid_points(x, y, z), **layer)
    return np.ascontiguousarray(E.reshape(len(z), len(y), len(x), 3).transpose(0, 3, 1, 2))


def planewaves(*, lam, sx, sy, gamma, zref, p, xyz, **_):
    """Plane-wave form (eq. 3 / eq. 9-10): E [n,3] complex128."""
    sx = np.ascontiguousarray(sx, dtype=np.float64)
    sy = np.ascontiguousarray(sy, dtype=np.float64)
    gamma = np.ascontiguousarray(gamma, dtype=np.complex128)
    zref = np.ascontiguousarray(zref, dtype=np.float64)
    assert p.dtype in (np.complex64, np.complex128) and p.flags.c_contiguous
    J = sx.shape[0]
    assert p.shape == (J, 3)
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    n = xyz.shape[0]
    E = np.zeros((n, 3), dtype=np.complex128)
    lib().scwo_planewaves(J, lam, _ptr(sx), _ptr(sy), _ptr(gamma), _ptr(zref), _ptr(p),
                          int(p.dtype == np.complex64), n, _ptr(xyz), _ptr(E))
    return E


# ----------------------------------------------------------------------------- Tier B
def _dirs(gamma, dir):
    if dir is not None:
        return np.where(np.asarray(dir) > 0, 1, -1)
    return np.where((gamma.imag > 0) | ((gamma.imag == 0) & (gamma.real >= 0)), 1, -1)


def tier_b_weights(*, lam, z_lo, z_hi, gamma, c=None, dir=None, z, **_):
    """g(z) of PAPER.md:430-432 times alpha: W[j,i] = c_j G(gamma_j, zref_j, z_i) (eq. 7, 30)."""
    gamma = np.asarray(gamma, dtype=np.complex128)
    zref = np.where(_dirs(gamma, dir) > 0, z_lo, z_hi)
    dz = np.asarray(z, dtype=np.float64)[None, :] - zref[:, None]
    W = np.exp(2j * np.pi * gamma[:, None] * dz / lam)
    if c is not None:
        W = W * np.asarray(c, dtype=np.complex128)[:, None]
    return W


def tier_b_spectra(*, U, Vn, V, z, **layer):
    """P(z) = [Q diag(alpha)] g(z): [3M, Fz] complex128, library matmul."""
    R = 3 * U * Vn
    W = tier_b_weights(z=z, **layer)
    Vm = V[:, :R].astype(np.complex128, copy=False).T      # [R, J] view of col-major storage
    return Vm @ W


def twiddles(n_freq, coords, period):
    """exp(i k s_u x) = exp(i 2 pi u x / X), u = -floor(n/2).. (eq. 6, eq. 10)."""
    u = np.arange(n_freq) - n_freq // 2
    t = np.outer(np.asarray(coords, dtype=np.float64) / period, u)
    t = t - np.rint(t)
    return np.exp(2j * np.pi * t)


def tier_b_synthesize(*, U, Vn, X, Y, P, x, y, **_):
    """eq. 10 on a rectilinear grid, separably: E_comp = F_x P_comp F_y^T -> [Fz,3,Ny,Nx]."""
    M = U * Vn
    Fz = P.shape[1]
    Fx = twiddles(U, x, X)            # [Nx, U]
    Fy = twiddles(Vn, y, Y)           # [Ny, Vn]
    E = np.empty((Fz, 3, len(y), len(x)), dtype=np.complex128)
    for i in range(Fz):
        for comp in range(3):
            Pc = P[comp * M:(comp + 1) * M, i].reshape(Vn, U)   # [v, u], u fastest
            E[i, comp] = Fy @ Pc @ Fx.T                          # [Ny, Nx]
    return E


def tier_b_grid(*, x, y, z, **layer):
    P = tier_b_spectra(z=z, **layer)
    return tier_b_synthesize(P=P, x=x, y=y, **layer)


def tier_b_points(*, U, Vn, X, Y, xyz, chunk=2048, **layer):
    """Factored evaluation at scattered points: P(z_p) per point, then the M-term sum."""
    M = U * Vn
    xyz = np.asarray(xyz, dtype=np.float64)
    E = np.empty((xyz.shape[0], 3), dtype=np.complex128)
    for s in range(0, xyz.shape[0], chunk):
        q = xyz[s:s + chunk]
        P = tier_b_spectra(U=U, Vn=Vn, z=q[:, 2], **layer)       # [3M, n]
        Fx = twiddles(U, q[:, 0], X)                               # [n, U]
        Fy = twiddles(Vn, q[:, 1], Y)                              # [n, Vn]
        T = (Fy[:, :, None] * Fx[:, None, :]).reshape(len(q), M)   # [n, m], u fastest
        for comp in range(3):
            E[s:s + chunk, comp] = np.einsum("nm,mn->n", T, P[comp * M:(comp + 1) * M])
    return E


# ----------------------------------------------------------------------------- exterior field (NEXT-1)
SIDE_ABOVE, SIDE_BELOW = 0, 1


def exterior_samples(*, side, U, Vn, X, Y, lam, n, z_face, p_face, z_inc=0.0, p_inc=None, xyz, **_):
    """Field outside the sample, eq. 9 then eq. 10, one frequency at a time -> E [n,3] complex128.

    above (z <= z_0):  p(s_m, z) = p_inc_m G[s_z(n), z_inc, z] + p_face_m G[-s_z(n), z_0, z]
    below (z >= z_L):  p(s_m, z) = p_face_m G[s_z(n), z_L, z]
    s_z by eq. 2 (Im >= 0), s_m = lam (u/X, v/Y) by eq. 6, G by eq. 7.  The reflected wave travels toward -z, hence
    -s_z (reading c-17).  p_face, p_inc: [M,3] complex.
    """
    xyz = np.asarray(xyz, dtype=np.float64)
    x, y, z = xyz[:, 0], xyz[:, 1], xyz[:, 2]
    k = 2.0 * np.pi / lam
    M = U * Vn
    p_face = np.asarray(p_face, dtype=np.complex128)
    p_inc = None if p_inc is None else np.asarray(p_inc, dtype=np.complex128)
    assert p_face.shape == (M, 3)
    E = np.zeros((xyz.shape[0], 3), dtype=np.complex128)
    for m in range(M):
        u, v = index_map(U, Vn, m)
        sx, sy = lam * u / X, lam * v / Y                                   # eq. 6
        s_z = sz(n, sx, sy)                                                 # eq. 2
        if side == SIDE_ABOVE:
            pz = p_face[m][None, :] * np.exp(1j * k * (z - z_face) * (-s_z))[:, None]       # reflected, eq. 7
            if p_inc is not None:
                pz = pz + p_inc[m][None, :] * np.exp(1j * k * (z - z_inc) * s_z)[:, None]  # incident
        else:
            pz = p_face[m][None, :] * np.exp(1j * k * (z - z_face) * s_z)[:, None]          # transmitted
        E += pz * np.exp(1j * k * (sx * x + sy * y))[:, None]               # eq. 10
    return E


def exterior_grid(*, x, y, z, **ext):
    """exterior_samples on a rectilinear grid -> E [Fz, 3, Ny, Nx] complex128 (planar layout)."""
    E = exterior_samples(xyz=grid_points(x, y, z), **ext)
    return np.ascontiguousarray(E.reshape(len(z), len(y), len(x), 3).transpose(0, 3, 1, 2))


# ----------------------------------------------------------------------------- detector intensity (NEXT-3)
def intensity(E):
    """I = |E_x|^2 + |E_y|^2 + |E_z|^2 from a planar field E [..., 3, Ny, Nx] -> [..., Ny, Nx] (the light intensity
    collected on a plane; reading c-18)."""
    E = np.asarray(E)
    return (E.real ** 2 + E.imag ** 2).sum(axis=-3)


def window_sum(I, window=None):
    """Detector window: S = sum of the intensity over the grid samples ix0 <= i < ix1, iy0 <= k < iy1 of every plane
    (plain sum over samples; "we detect the intensity of the transmission waves", 554).  I [..., Ny, Nx]."""
    I = np.asarray(I, dtype=np.float64)
    if window is None:
        return I.sum(axis=(-2, -1))
    ix0, ix1, iy0, iy1 = window
    return I[..., iy0:iy1, ix0:ix1].sum(axis=(-2, -1))


def absorbance(S, S0):
    """A = -log10(S / S0): absorbance of a detector reading against a reference reading (Fig. 6)."""
    return -np.log10(np.asarray(S, dtype=np.float64) / np.asarray(S0, dtype=np.float64))


def band_absorbance(S, S0, w=None):
    """Absorbance of a whole band: -log10(sum_i w_i S_i / sum_i w_i S0_i), spectral weights w (None = ones)."""
    S, S0 = np.asarray(S, dtype=np.float64), np.asarray(S0, dtype=np.float64)
    w = np.ones_like(S) if w is None else np.asarray(w, dtype=np.float64)
    return float(-np.log10((w * S).sum() / (w * S0).sum()))


# ----------------------------------------------------------------------------- V builder (NEXT-2, eq. 33)
def wrap_index(U, Vn, m, mp):
    """m (-) m': index of the frequency (u - u', v - v') wrapped back onto the U x Vn grid of eq. 6 (DESIGN.md reading
    c-20: the "m - m'" of eq. 33 is a difference of frequency VECTORS, and the circulant of eq. 21, PAPER.md:198-212,
    wraps it per axis -- a block-circulant matrix with circulant blocks)."""
    u, v = index_map(U, Vn, m)
    up, vp = index_map(U, Vn, mp)
    du = (u - up + U // 2) % U - U // 2
    dv = (v - vp + Vn // 2) % Vn - Vn // 2
    return (dv + Vn // 2) * U + du + U // 2


def build_V(*, U, Vn, X, Y, lam, Q, psi, alpha=None):
    """V = T Q [diag(alpha)]: the map from the eigenvector matrix Q [J, ldQ >= 4M] (column-major
    [4M x J], rows P_x, P_y, B_x, B_y in blocks of M, eq. 19-20) to the plane-wave amplitudes [P_x; P_y; P_z]:
    the P_x, P_y rows are copied, and eq. 33 gives the z component,

        [P_z]_m = + sum_{m'} psi_{m'} { [s_y]_{m-m'} [b_x]_{m-m'} - [s_x]_{m-m'} [b_y]_{m-m'} },

    one (m, m') term at a time.  Sign: + (reading c-19: the printed minus comes from a curl written with the opposite sign
    at PAPER.md:344 and breaks s.p = 0, eq. 14); psi_m are the Fourier-series coefficients of 1/n^2 on the grid of eq. 6,
    1/n^2(r) = sum_m psi_m exp(ik s_m.r) (reading c-21), s_m = lam (u/X, v/Y).  Returns V [J, 3M] (column-major [3M x J])."""
    M = U * Vn
    Q = np.asarray(Q)
    J = Q.shape[0]
    psi = np.asarray(psi, dtype=np.complex128)
    assert Q.shape[1] >= 4 * M and psi.shape == (M,)
    Qc = Q[:, :4 * M].astype(np.complex128)
    sx = np.empty(M)
    sy = np.empty(M)
    for m in range(M):
        u, v = index_map(U, Vn, m)
        sx[m], sy[m] = lam * u / X, lam * v / Y                      # eq. 6
    q = sy[None, :] * Qc[:, 2 * M:3 * M] - sx[None, :] * Qc[:, 3 * M:4 * M]       # [J, M]: s_y b_x - s_x b_y per column
    V = np.zeros((J, 3 * M), dtype=np.complex128)
    V[:, :2 * M] = Qc[:, :2 * M]
    for m in range(M):
        for mp in range(M):
            V[:, 2 * M + m] += psi[mp] * q[:, wrap_index(U, Vn, m, mp)]
    if alpha is not None:
        V *= np.asarray(alpha, dtype=np.complex128)[:, None]
    return V


# ----------------------------------------------------------------------------- alpha propagation (NEXT-4, eq. 24-26)
def interface_factors(*, lam, z_a, z_b, gamma, dir=None):
    """Diagonals of the two interface matrices of a layer between z_a = z_{l-1} and z_b = z_l (symbols
    de-garbled per reading c-7):  Q'_l = Qcheck + Qhat G(Gamma, z_l, z_{l-1}) = Q diag(d_acute),
                                   Q`_l = Qcheck G(Gamma, z_{l-1}, z_l) + Qhat = Q diag(d_grave),
    Qcheck / Qhat = the "+" / "-" columns of Q, G of eq. 7.  Every exponential decays (reading c-1)."""
    gamma = np.asarray(gamma, dtype=np.complex128)
    plus = _dirs(gamma, dir) > 0
    d_acute = np.where(plus, 1.0, np.array([green(g, z_b, z_a, lam) for g in gamma]))
    d_grave = np.where(plus, np.array([green(g, z_a, z_b, lam) for g in gamma]), 1.0)
    return d_acute, d_grave


def propagate_alpha(*, lam, z_if, Q, gamma, dir=None, r0):
    """alpha^(l) of every layer from the field vector r0 = Gbar Rbar + Rhat at the top interface z_0 (eq. 24,
    PAPER.md:254-256) through the middle-boundary conditions (eq. 25):
        alpha^(1) = Q'_1^-1 r0,      alpha^(l) = Q'_l^-1 Q`_{l-1} alpha^(l-1),
    and the field vector at the bottom interface, Rcheck = Q`_L alpha^(L) (eq. 26).  The linear solve is a library routine
    (numpy / LAPACK).  Q: list of L arrays [n, n] in MATHEMATICAL orientation (row = field component, column = mode),
    gamma: list of [n], dir: list of [n] or None.  Returns (list of alpha [n], r_L)."""
    r = np.asarray(r0, dtype=np.complex128)
    alphas = []
    for l in range(len(Q)):
        Ql = np.asarray(Q[l], dtype=np.complex128)
        d_acute, d_grave = interface_factors(lam=lam, z_a=z_if[l], z_b=z_if[l + 1], gamma=gamma[l],
                                             dir=None if dir is None else dir[l])
        Q_acute = Ql * d_acute[None, :]
        alpha = np.linalg.solve(Q_acute, r)
        alphas.append(alpha)
        r = (Ql * d_grave[None, :]) @ alpha
    return alphas, r

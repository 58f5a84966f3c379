"""Seeded synthetic inputs for the sCWatter field-evaluation hot path.

This module serves both the oracle and the CUDA path with *data* (numpy arrays and
python scalars); it contains no field-evaluation arithmetic and imports neither side.
The recipe takes the shapes of BASELINE.json's
five configs: M = U*V spatial frequencies on the grid of eq. 6, J = 4M
modes per layer in the paper's interleave j = 4 m + 2 pol + d, d = 0 "+", d = 1 "-"
(PAPER.md:220, 246), eigenvector columns V[3M x J] (column-major), coefficients c_j,
signed z-wavenumbers gamma_j = +-sqrt(n_j^2 - |s_m|^2) (eq. 2 shape, Im >= 0 branch).
The paper's own sample images are not available; these inputs stand in for them.

RNG: numpy Generator(Philox(key=[7293, id])),
id = config*2^20 + lambda_index*2^8 + layer*2^3 + array,
array: 0 n_j, 1 V, 2 c, 3 thickness, 4 points, 5 oracle subset, 6 evanescent mask/sigma, 7 exterior amplitudes.
"""
from dataclasses import dataclass

import numpy as np

A_N, A_V, A_C, A_T, A_PTS, A_SUB, A_EVAN, A_EXT = range(8)


def rng(config: int, array: int, lam_index: int = 0, layer: int = 0) -> np.random.Generator:
    ident = config * 2**20 + lam_index * 2**8 + layer * 2**3 + array
    return np.random.Generator(np.random.Philox(key=[7293, ident]))


@dataclass(frozen=True)
class Config:
    cid: int
    name: str
    U: int
    Vn: int
    L: float                 # patch size X = Y = L (same unit as lambda)
    lams: tuple              # vacuum wavelengths
    n_layers: int
    planes: int              # z-planes per layer
    Nx: int
    Ny: int
    dtypes: tuple            # numpy complex dtypes the config is run in
    eta: float = 0.05        # Im n_j ~ U[0, eta]
    evanescent: float = 0.0  # fraction of modes given |s| ~ U[Re n, 2 Re n]
    thickness: tuple = (1.0, 3.0)   # layer thickness ~ U[lo, hi] (or fixed if lo == hi)
    n_points: int = 0        # scattered points (point-path configs)


CONFIGS = {
    0: Config(0, "toy 9x9", 9, 9, 8.0, (1.0,), 1, 16, 64, 64, (np.complex128,),
              thickness=(2.0, 2.0)),
    1: Config(1, "slab stack 33x33", 33, 33, 32.0, (1.0,), 4, 64, 256, 256,
              (np.complex64, np.complex128)),
    2: Config(2, "large patch 65x65", 65, 65, 64.0, (1.0,), 2, 16, 512, 512,
              (np.complex64,), eta=0.1, evanescent=0.25),
    3: Config(3, "scattered points 33x33", 33, 33, 32.0, (1.0,), 1, 0, 0, 0,
              (np.complex64,), thickness=(2.0, 2.0), n_points=4_000_000),
    4: Config(4, "spectroscopy sweep 17x17", 17, 17, 16.0,
              tuple(np.linspace(0.5, 1.5, 32).tolist()), 2, 16, 256, 256,
              (np.complex64,)),
}


def _sqrt_upper(a):
    """Principal square root moved to the closed upper half plane (Im >= 0; Re >= 0 on the axis)."""
    a = np.asarray(a, dtype=np.complex128)
    a = a.real + 1j * np.where(a.imag == 0.0, 0.0, a.imag)       # drop -0.0
    g = np.sqrt(a)
    flip = (g.imag < 0) | ((g.imag == 0) & (g.real < 0))
    return np.where(flip, -g, g)


def freq_uv(U: int, Vn: int):
    """Integer frequencies (u_m, v_m) for m = 0..M-1, u fastest."""
    m = np.arange(U * Vn)
    return m % U - U // 2, m // U - Vn // 2


def stack_interfaces(cfg: Config):
    """z_0 = 0, z_l = z_{l-1} + t_l; thicknesses are fixed across wavelengths."""
    z = [0.0]
    for layer in range(cfg.n_layers):
        lo, hi = cfg.thickness
        t = lo if lo == hi else float(rng(cfg.cid, A_T, 0, layer).uniform(lo, hi))
        z.append(z[-1] + t)
    return np.array(z)


def grid_coords(cfg: Config, layer: int, planes=None, Nx=None, Ny=None):
    """x_i = i X/Nx, y_k = k Y/Ny (one period, endpoint excluded), z cell-centred in the layer."""
    zi = stack_interfaces(cfg)
    Fz = cfg.planes if planes is None else planes
    Nx = cfg.Nx if Nx is None else Nx
    Ny = cfg.Ny if Ny is None else Ny
    x = np.arange(Nx) * (cfg.L / Nx)
    y = np.arange(Ny) * (cfg.L / Ny)
    z = zi[layer] + (np.arange(Fz) + 0.5) * ((zi[layer + 1] - zi[layer]) / Fz)
    return x, y, z


def make_layer(cfg: Config, layer: int = 0, lam_index: int = 0, dtype=np.complex128,
               ldV=None, with_V=True):
    """One layer at one wavelength as a dict of arrays (see oracle/__init__.py for the keys)."""
    U, Vn = cfg.U, cfg.Vn
    M = U * Vn
    J = 4 * M
    R = 3 * M
    lam = float(cfg.lams[lam_index])
    zi = stack_interfaces(cfg)

    g = rng(cfg.cid, A_N, lam_index, layer)
    n = g.uniform(1.3, 1.6, J) + 1j * g.uniform(0.0, cfg.eta, J)
    u, v = freq_uv(U, Vn)
    mj = np.arange(J) // 4
    s2 = (lam * u[mj] / cfg.L) ** 2 + (lam * v[mj] / cfg.L) ** 2
    if cfg.evanescent > 0:
        ge = rng(cfg.cid, A_EVAN, lam_index, layer)
        mask = ge.uniform(0, 1, J) < cfg.evanescent
        sigma = ge.uniform(n.real, 2 * n.real)
        s2 = np.where(mask, sigma**2, s2)
    dirs = np.where(np.arange(J) % 2 == 0, 1, -1).astype(np.int8)
    gamma = dirs * _sqrt_upper(n * n - s2)

    gc = rng(cfg.cid, A_C, lam_index, layer)
    c = ((gc.standard_normal(J) + 1j * gc.standard_normal(J)) / np.sqrt(2.0)).astype(dtype)

    out = dict(U=U, Vn=Vn, X=cfg.L, Y=cfg.L, lam=lam, z_lo=float(zi[layer]),
               z_hi=float(zi[layer + 1]), gamma=gamma, c=c, dir=dirs, J=J)
    if with_V:
        ldV = R if ldV is None else ldV
        fdt = np.float32 if dtype == np.complex64 else np.float64
        gv = rng(cfg.cid, A_V, lam_index, layer)
        Vs = np.zeros((J, ldV), dtype=dtype)          # column-major [ldV x J]
        scale = 1.0 / np.sqrt(2.0 * M)
        step = max(1, (1 << 24) // R)                 # generate in column chunks (memory)
        for j0 in range(0, J, step):
            j1 = min(J, j0 + step)
            blk = gv.standard_normal((j1 - j0, R, 2)) * scale
            Vs[j0:j1, :R] = (blk[..., 0] + 1j * blk[..., 1]).astype(dtype)
        assert Vs.view(fdt).shape == (J, 2 * ldV)
        out["V"] = Vs
    return out


def make_planewaves(cfg: Config, layer: int = 0, lam_index: int = 0, dtype=np.complex64):
    """Plane-wave mode table for the point path (config 3): one plane wave per mode j."""
    lay = make_layer(cfg, layer, lam_index, dtype=np.complex128, with_V=False)
    U, Vn = cfg.U, cfg.Vn
    M = U * Vn
    J = 4 * M
    u, v = freq_uv(U, Vn)
    mj = np.arange(J) // 4
    lam = lay["lam"]
    sx = lam * u[mj] / cfg.L
    sy = lam * v[mj] / cfg.L
    gp = rng(cfg.cid, A_V, lam_index, layer)
    p = ((gp.standard_normal((J, 3)) + 1j * gp.standard_normal((J, 3)))
         / np.sqrt(2.0 * M)).astype(dtype)
    zref = np.where(lay["dir"] > 0, lay["z_lo"], lay["z_hi"]).astype(np.float64)
    return dict(lam=lam, sx=sx, sy=sy, gamma=lay["gamma"], zref=zref, p=p, J=J,
                z_lo=lay["z_lo"], z_hi=lay["z_hi"])


N_ABOVE, N_BELOW = 1.0, 1.5          # config 0's half-spaces (BASELINE.json configs[0]); used for every config


def make_exterior(cfg: Config, side: int, lam_index: int = 0, dtype=np.complex64, z_inc=None):
    """Exterior-field inputs (eq. 9): side 0 = above the stack (incident + reflected amplitudes, n = 1.0),
    side 1 = below (transmitted amplitudes, n = 1.5).  Amplitudes are complex normals / sqrt(M) per component;
    the incident wave is referenced one wavelength above z_0 unless z_inc is given."""
    U, Vn = cfg.U, cfg.Vn
    M = U * Vn
    lam = cfg.lams[lam_index]
    zi = stack_interfaces(cfg)
    g = rng(cfg.cid, A_EXT, lam_index, side)
    draw = lambda: ((g.standard_normal((M, 3)) + 1j * g.standard_normal((M, 3))) / np.sqrt(2.0 * M)).astype(dtype)
    d = dict(side=side, U=U, Vn=Vn, X=cfg.L, Y=cfg.L, lam=lam, p_face=draw())
    if side == 0:
        d.update(n=complex(N_ABOVE), z_face=float(zi[0]), z_inc=float(zi[0] - lam if z_inc is None else z_inc), p_inc=draw())
    else:
        d.update(n=complex(N_BELOW), z_face=float(zi[-1]))
    return d


def make_points(cfg: Config, n=None, layer: int = 0):
    """Scattered points r ~ U[0,L)^2 x [z_lo, z_hi) as [n,3] float64."""
    n = cfg.n_points if n is None else n
    zi = stack_interfaces(cfg)
    g = rng(cfg.cid, A_PTS, 0, layer)
    xyz = np.empty((n, 3))
    xyz[:, 0] = g.uniform(0.0, cfg.L, n)
    xyz[:, 1] = g.uniform(0.0, cfg.L, n)
    xyz[:, 2] = g.uniform(zi[layer], zi[layer + 1], n)
    return xyz


def sample_subset(cfg: Config, n_total: int, n_pick: int, lam_index: int = 0, layer: int = 0):
    """Seeded subset of flat output-sample indices for sampled parity checks."""
    g = rng(cfg.cid, A_SUB, lam_index, layer)
    return np.sort(g.choice(n_total, size=min(n_pick, n_total), replace=False))

"""alpha propagation across layers (eq. 24-26): oracle pins (CPU) and GPU parity through the C ABI.

Pins of oracle.propagate_alpha: the interface matrices written out as the paper defines them (Qcheck + Qhat G, ...) must
make both sides of eq. 25 equal; a stack of identical layers propagates every mode analytically; a single layer equals
the explicit inverse; the solve against a pure-python Gaussian elimination on a tiny system.
"""
import cmath
import math

import numpy as np
import pytest

import oracle


def random_stack(n, L, seed, dtype=np.complex128, lam=0.8):
    g = np.random.default_rng(seed)
    z_if = np.concatenate([[0.0], np.cumsum(g.uniform(0.3, 0.9, L))])
    Q, gamma, dirs = [], [], []
    for _ in range(L):
        A = (g.standard_normal((n, n)) + 1j * g.standard_normal((n, n))) / np.sqrt(2 * n)
        Q.append((A + 1.5 * np.eye(n)).astype(dtype))                       # well conditioned, not diagonally trivial
        d = np.where(np.arange(n) % 2 == 0, 1, -1).astype(np.int8)
        gamma.append(d * (g.uniform(0.2, 1.4, n) + 1j * g.uniform(0.0, 0.4, n)))
        dirs.append(d)
    r0 = ((g.standard_normal(n) + 1j * g.standard_normal(n)) / np.sqrt(2)).astype(dtype)
    return dict(lam=lam, z_if=z_if, Q=Q, gamma=gamma, dir=dirs, r0=r0)


def test_middle_boundary_condition_with_the_papers_matrices():
    """Eq. 25 with Q'_l and Q`_l assembled exactly as printed: Qcheck, Qhat by column parity, G of
    eq. 7 as full diagonal matrices."""
    st = random_stack(12, 3, seed=1)
    alphas, rL = oracle.propagate_alpha(**st)
    k = 2 * math.pi / st["lam"]
    def mats(l):
        Q, gam = st["Q"][l], st["gamma"][l]
        plus = np.arange(12) % 2 == 0
        Qc, Qh = Q * plus[None, :], Q * (~plus)[None, :]
        za, zb = st["z_if"][l], st["z_if"][l + 1]
        G_ba = np.diag(np.exp(1j * k * (za - zb) * gam))                    # G(Gamma, z_l, z_{l-1})
        G_ab = np.diag(np.exp(1j * k * (zb - za) * gam))                    # G(Gamma, z_{l-1}, z_l)
        return Qc + Qh @ G_ba, Qc @ G_ab + Qh
    Qa1, _ = mats(0)
    assert np.abs(Qa1 @ alphas[0] - st["r0"]).max() < 1e-13                 # eq. 24
    for l in (1, 2):
        Qa, _ = mats(l)
        _, Qg_prev = mats(l - 1)
        assert np.abs(Qg_prev @ alphas[l - 1] - Qa @ alphas[l]).max() < 1e-12      # eq. 25
    assert np.abs(mats(2)[1] @ alphas[2] - rL).max() < 1e-13                # eq. 26


def test_identical_layers_propagate_analytically():
    """Same Q, Gamma in consecutive layers: alpha^(l)_j = G(gamma_j, z_{l-2}, z_{l-1}) alpha^(l-1)_j for "+" modes and
    alpha^(l-1)_j = G(Gamma_j, z_l, z_{l-1}) alpha^(l)_j for "-" modes (every mode just propagates, eq. 23)."""
    st = random_stack(10, 1, seed=2)
    z_if = np.array([0.0, 0.4, 1.1, 1.5])
    st3 = dict(st, z_if=z_if, Q=st["Q"] * 3, gamma=st["gamma"] * 3, dir=st["dir"] * 3)
    alphas, _ = oracle.propagate_alpha(**st3)
    k = 2 * math.pi / st["lam"]
    gam = st["gamma"][0]
    for l in (1, 2):
        t_prev, t_cur = z_if[l] - z_if[l - 1], z_if[l + 1] - z_if[l]
        for j in range(10):
            if j % 2 == 0:
                ref = cmath.exp(1j * k * gam[j] * t_prev) * alphas[l - 1][j]
            else:
                ref = alphas[l - 1][j] / cmath.exp(1j * k * (-t_cur) * gam[j])
            assert abs(alphas[l][j] - ref) < 1e-11 * max(1.0, abs(ref))


def test_single_layer_is_the_explicit_inverse_and_gauss():
    st = random_stack(6, 1, seed=3)
    alphas, _ = oracle.propagate_alpha(**st)
    d_acute, _ = oracle.interface_factors(lam=st["lam"], z_a=0.0, z_b=st["z_if"][1], gamma=st["gamma"][0], dir=st["dir"][0])
    Qa = st["Q"][0] * d_acute[None, :]
    assert np.abs(np.linalg.inv(Qa) @ st["r0"] - alphas[0]).max() < 1e-12
    # pure-python Gaussian elimination with partial pivoting
    A = [[complex(v) for v in row] for row in Qa]
    b = [complex(v) for v in st["r0"]]
    n = 6
    for c in range(n):
        p = max(range(c, n), key=lambda r: abs(A[r][c]))
        A[c], A[p], b[c], b[p] = A[p], A[c], b[p], b[c]
        for r in range(c + 1, n):
            f = A[r][c] / A[c][c]
            for cc in range(c, n):
                A[r][cc] -= f * A[c][cc]
            b[r] -= f * b[c]
    xs = [0j] * n
    for r in range(n - 1, -1, -1):
        xs[r] = (b[r] - sum(A[r][cc] * xs[cc] for cc in range(r + 1, n))) / A[r][r]
    assert np.abs(np.array(xs) - alphas[0]).max() < 1e-12
    # |d| <= 1: every interface factor decays (reading c-1)
    da, dg = oracle.interface_factors(lam=st["lam"], z_a=0.0, z_b=st["z_if"][1], gamma=st["gamma"][0], dir=None)
    assert np.abs(da).max() <= 1 + 1e-15 and np.abs(dg).max() <= 1 + 1e-15


# ------------------------------------------------------------------------------------------------ GPU
def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.gpu
@pytest.mark.parametrize("dtype,tol", [(np.complex64, 2e-4), (np.complex128, 1e-10)])
@pytest.mark.parametrize("n,L,with_dir", [(4, 1, True), (36, 3, True), (100, 2, False), (324, 3, True), (517, 2, True)])
def test_propagate_alpha_against_the_oracle(dtype, tol, n, L, with_dir):
    """scw_propagate_alpha (blocked LU on the GPU) against oracle.propagate_alpha (LAPACK): every alpha of every layer and
    the bottom field vector; n not a multiple of the 64-column panel, one to several panels, dir given or derived."""
    import torch
    import paper_2404_07293_b200 as scw
    st = random_stack(n, L, seed=n + L, dtype=dtype)
    ref_a, ref_r = oracle.propagate_alpha(lam=st["lam"], z_if=st["z_if"], Q=st["Q"], gamma=st["gamma"],
                                          dir=st["dir"] if with_dir else None, r0=st["r0"])
    ctx = scw.Context(0)
    try:
        # the C ABI takes column-major Q: tensor row j = column j of the mathematical matrix
        Qd = [dev(np.ascontiguousarray(q.T)) for q in st["Q"]]
        alphas, rL = scw.scw_propagate_alpha(ctx, lam=st["lam"], z_if=st["z_if"], Q=Qd, gamma=[dev(g) for g in st["gamma"]],
                                             dir=[dev(d) for d in st["dir"]] if with_dir else None, r0=dev(st["r0"]))
        torch.cuda.synchronize()
        for l in range(L):
            assert np.abs(alphas[l].cpu().numpy() - ref_a[l]).max() / np.abs(ref_a[l]).max() <= tol, l
        assert np.abs(rL.cpu().numpy() - ref_r).max() / np.abs(ref_r).max() <= tol
    finally:
        ctx.close()


@pytest.mark.gpu
def test_propagate_alpha_config1_size():
    """n = 4M = 4356 (config 1), two layers, complex128: 69 panels, trailing updates on the DMMA kernel."""
    import torch
    import paper_2404_07293_b200 as scw
    st = random_stack(4356, 2, seed=5)
    ref_a, ref_r = oracle.propagate_alpha(**st)
    ctx = scw.Context(0)
    try:
        Qd = [dev(np.ascontiguousarray(q.T)) for q in st["Q"]]
        alphas, rL = scw.scw_propagate_alpha(ctx, lam=st["lam"], z_if=st["z_if"], Q=Qd, gamma=[dev(g) for g in st["gamma"]],
                                             dir=[dev(d) for d in st["dir"]], r0=dev(st["r0"]))
        torch.cuda.synchronize()
        for l in range(2):
            assert np.abs(alphas[l].cpu().numpy() - ref_a[l]).max() / np.abs(ref_a[l]).max() <= 1e-10
        assert np.abs(rL.cpu().numpy() - ref_r).max() / np.abs(ref_r).max() <= 1e-10
    finally:
        ctx.close()


# ------------------------------------------------------------------------------------------------ pivoting
def rows_moved(A):
    """How many rows LAPACK's partial pivoting (same |re| + |im| measure as the GPU kernel) exchanges on A."""
    import scipy.linalg
    _, piv = scipy.linalg.lu_factor(A)
    return int((piv != np.arange(len(piv))).sum())


def pivoting_stack(kind, n, L, seed, dtype):
    """Stacks whose Q'_l = Q diag(d_acute) are NOT diagonally dominant (an eigenvector matrix is not), so
    the LU of eq. 24-25 has to exchange rows:
      gauss  -- plain complex Gaussian Q, no dominant diagonal at all;
      perm   -- the well-conditioned stack of random_stack with its rows permuted;
      last   -- 1.5 x (cyclic shift by n - 8 rows) + noise: the largest entry of every column sits in the last 8 rows of the
                matrix for every column, i.e. always in the rows of the last CTA of the panel kernel;
      ties   -- gauss with pairs of candidates of exactly equal |re| + |im| in many columns (3 and 3i; 2 + 1i and 1 + 2i)."""
    st = random_stack(n, L, seed, dtype=dtype)
    g = np.random.default_rng(seed + 1000)
    for l in range(L):
        if kind in ("gauss", "ties"):
            A = (g.standard_normal((n, n)) + 1j * g.standard_normal((n, n))) / np.sqrt(2)
            if kind == "ties":
                for c in range(0, n, 3):
                    r1, r2 = g.choice(n, 2, replace=False)
                    A[r1, c], A[r2, c] = (3.0, 3.0j) if c % 2 else (2.0 + 1.0j, 1.0 + 2.0j)
        elif kind == "perm":
            A = st["Q"][l].astype(np.complex128)[g.permutation(n)]
        elif kind == "last":
            A = (g.standard_normal((n, n)) + 1j * g.standard_normal((n, n))) / np.sqrt(2 * n)
            s = n - min(8, n // 2)
            A[(np.arange(n) + s) % n, np.arange(n)] += 1.5
        st["Q"][l] = A.astype(dtype)
    return st


@pytest.mark.gpu
@pytest.mark.parametrize("dtype,tol", [(np.complex64, 2e-4), (np.complex128, 1e-10)])
@pytest.mark.parametrize("kind,n,L", [("gauss", 36, 3), ("gauss", 324, 2), ("gauss", 517, 2), ("perm", 324, 3), ("perm", 517, 2),
                                      ("last", 100, 2), ("last", 517, 2), ("ties", 36, 2), ("ties", 324, 2)])
def test_propagate_alpha_with_row_exchanges(kind, dtype, tol, n, L):
    """The LU behind eq. 24-25 on matrices that need partial pivoting: LAPACK exchanges more
    than a quarter of the rows on every Q'_l here (asserted), so the cross-CTA pivot search, the candidate-row exchange,
    k_lu_laswp and k_lu_apply_piv all run.  The SOLUTION is compared, not the permutation.  Tolerance: the usual
    1e-10 / 2e-4 of max|alpha|, not widened: both sides solve in fp64 from the same rounded inputs with the same pivoting
    measure, and the measured differences stay below 1e-12 up to prod_l cond_2(Q'_l) = 2e7 (asserted < 1e8 here so that
    eps cond stays well inside the tolerance)."""
    import torch
    import paper_2404_07293_b200 as scw
    st = pivoting_stack(kind, n, L, seed=7 * n + L, dtype=dtype)
    ref_a, ref_r = oracle.propagate_alpha(**st)
    cond = 1.0
    for l in range(L):
        d_acute, _ = oracle.interface_factors(lam=st["lam"], z_a=st["z_if"][l], z_b=st["z_if"][l + 1], gamma=st["gamma"][l],
                                              dir=st["dir"][l])
        Qa = st["Q"][l].astype(np.complex128) * d_acute[None, :]
        assert rows_moved(Qa) > n // 4, (kind, l)
        cond *= np.linalg.cond(Qa)
    assert cond < 1e8
    ctx = scw.Context(0)
    try:
        Qd = [dev(np.ascontiguousarray(q.T)) for q in st["Q"]]
        alphas, rL = scw.scw_propagate_alpha(ctx, lam=st["lam"], z_if=st["z_if"], Q=Qd, gamma=[dev(g) for g in st["gamma"]],
                                             dir=[dev(d) for d in st["dir"]], r0=dev(st["r0"]))
        torch.cuda.synchronize()
        for l in range(L):
            assert np.abs(alphas[l].cpu().numpy() - ref_a[l]).max() / np.abs(ref_a[l]).max() <= tol, (l, cond)
        assert np.abs(rL.cpu().numpy() - ref_r).max() / np.abs(ref_r).max() <= tol
    finally:
        ctx.close()


@pytest.mark.gpu
def test_propagate_alpha_config1_size_with_row_exchanges():
    """n = 4356 (config 1), complex128, plain Gaussian Q: 69 panels that all pivot across CTAs."""
    import torch
    import paper_2404_07293_b200 as scw
    n = 4356
    st = pivoting_stack("gauss", n, 1, seed=11, dtype=np.complex128)
    ref_a, ref_r = oracle.propagate_alpha(**st)
    d_acute, _ = oracle.interface_factors(lam=st["lam"], z_a=st["z_if"][0], z_b=st["z_if"][1], gamma=st["gamma"][0], dir=st["dir"][0])
    Qa = st["Q"][0] * d_acute[None, :]
    assert rows_moved(Qa) > n // 4
    tol = 1e-10
    ctx = scw.Context(0)
    try:
        alphas, rL = scw.scw_propagate_alpha(ctx, lam=st["lam"], z_if=st["z_if"], Q=[dev(np.ascontiguousarray(st["Q"][0].T))],
                                             gamma=[dev(st["gamma"][0])], dir=[dev(st["dir"][0])], r0=dev(st["r0"]))
        torch.cuda.synchronize()
        err = np.abs(alphas[0].cpu().numpy() - ref_a[0]).max() / np.abs(ref_a[0]).max()
        assert err <= tol, (err, tol)
        assert np.abs(rL.cpu().numpy() - ref_r).max() / np.abs(ref_r).max() <= tol
    finally:
        ctx.close()


@pytest.mark.gpu
@pytest.mark.parametrize("kind", ["zero_column", "nan_entry", "zero_matrix"])
def test_propagate_alpha_singular_or_nan_Q_gives_non_finite_alpha_and_a_healthy_ctx(kind):
    """An exactly singular Q (a zero column: a zero pivot, then 0/0 = NaN below it, then columns without any finite pivot
    candidate) or a Q holding NaN: alpha comes back non-finite, no error, no fault -- and the same ctx then solves a
    regular stack correctly (include/scwatter.h: 'the ctx and the device stay usable')."""
    import torch
    import paper_2404_07293_b200 as scw
    n = 200
    st = random_stack(n, 2, seed=21)
    bad = dict(st, Q=[q.copy() for q in st["Q"]])
    if kind == "zero_column":
        bad["Q"][0][:, 70] = 0.0
    elif kind == "nan_entry":
        bad["Q"][0][130, 5] = np.nan
    else:
        bad["Q"][0][:] = 0.0
    ctx = scw.Context(0)
    try:
        def run(s):
            out = scw.scw_propagate_alpha(ctx, lam=s["lam"], z_if=s["z_if"], Q=[dev(np.ascontiguousarray(q.T)) for q in s["Q"]],
                                          gamma=[dev(g) for g in s["gamma"]], dir=[dev(d) for d in s["dir"]], r0=dev(s["r0"]))
            torch.cuda.synchronize()
            return out
        alphas, _ = run(bad)
        assert not np.isfinite(alphas[0].cpu().numpy()).all()
        ref_a, ref_r = oracle.propagate_alpha(**st)
        alphas, rL = run(st)
        for l in range(2):
            assert np.abs(alphas[l].cpu().numpy() - ref_a[l]).max() / np.abs(ref_a[l]).max() <= 1e-10
        assert np.abs(rL.cpu().numpy() - ref_r).max() / np.abs(ref_r).max() <= 1e-10
    finally:
        ctx.close()

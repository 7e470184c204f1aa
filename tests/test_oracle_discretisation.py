"""Pins of the oracle's building blocks against what the paper and the mathematics fix
(SURVEY.md 8(c.3) P1-P4).  CPU only."""
import math

import numpy as np
import pytest

from oracle import dlr_oracle as O
from paper_2110_13481_b200 import inputs


def grids(cfg):
    gx = O.Grid3((cfg["n_x"],) * 3, (cfg["x_lo"],) * 3, (cfg["x_hi"],) * 3)
    gv = O.Grid3((cfg["n_v"],) * 3, (cfg["v_lo"],) * 3, (cfg["v_hi"],) * 3)
    return gx, gv


# ---------------- P1: DFT convention (R3) against the naive O(n^2) definition ----------------
@pytest.mark.parametrize("n", [4, 8, 16])
def test_fft3_matches_naive_dft(n):
    rng = np.random.default_rng(n)
    A = rng.standard_normal((2, n, n, n))
    j = np.arange(n)
    W = np.exp(-2j * math.pi * np.outer(j, j) / n)          # forward kernel e^{-2 pi i m j/n}
    naive = np.einsum("ai,bj,ck,rijk->rabc", W, W, W, A)
    assert np.abs(O.fft3(A) - naive).max() <= 1e-12 * np.abs(naive).max()
    assert np.abs(O.ifft3(O.fft3(A)).real - A).max() <= 1e-13
    # Parseval with the unnormalised forward transform
    assert abs(np.sum(np.abs(O.fft3(A)) ** 2) / n ** 3 - np.sum(A * A)) <= 1e-10 * np.sum(A * A)


def test_fft_of_cosine_is_two_spikes_and_axis_order():
    """axis convention: x1 is the fastest (last numpy) axis; cos(2 pi m x1 / L) -> spikes at +-m on that axis"""
    g = O.Grid3((8, 4, 4), (0, 0, 0), (4 * math.pi, 1.0, 1.0))
    A = np.broadcast_to(np.cos(0.5 * g.coord(0)), g.shape)[None]       # k = 0.5 = 2 pi * 1 / (4 pi)
    Ah = O.fft3(A)[0]
    expect = np.zeros(g.shape, dtype=complex)
    expect[0, 0, 1] = expect[0, 0, 7] = 0.5 * g.N
    assert np.abs(Ah - expect).max() < 1e-10


def test_wavenumbers_and_nyquist():
    g = O.Grid3((8, 8, 8), (0,) * 3, (4 * math.pi,) * 3)
    assert list(g.m(0)) == [0, 1, 2, 3, -4, -3, -2, -1]
    assert g.kt(0).reshape(-1)[4] == 0.0 and abs(g.k(0).reshape(-1)[4]) == pytest.approx(2.0)
    # derivative of sin(x1/2) is cos(x1/2)/2, exact for a resolved mode
    A = np.broadcast_to(np.sin(0.5 * g.coord(0)), g.shape)[None]
    assert np.abs(O.deriv(A, g, 0)[0] - 0.5 * np.cos(0.5 * g.coord(0))).max() < 1e-13
    # the spectral derivative matrix is exactly skew: <A, dB> = -<dA, B>
    rng = np.random.default_rng(0)
    A, B = rng.standard_normal((2, 1, 8, 8, 8))
    for d in range(3):
        assert abs(np.sum(A * O.deriv(B, g, d)) + np.sum(O.deriv(A, g, d) * B)) < 1e-11


# ---------------- P2: small dense ----------------
@pytest.mark.parametrize("n", [3, 10, 20])
def test_jacobi(n):
    rng = np.random.default_rng(n)
    M = rng.standard_normal((n, n))
    M = M + M.T
    lam, T = O.jacobi_eigh(M)
    assert np.abs(T @ np.diag(lam) @ T.T - M).max() < 1e-13 * n
    assert np.abs(T.T @ T - np.eye(n)).max() < 1e-13
    assert np.abs(np.sort(lam) - np.linalg.eigvalsh(M)).max() < 1e-12


def test_jacobi_degenerate():
    rng = np.random.default_rng(1)
    Q, _ = np.linalg.qr(rng.standard_normal((12, 12)))
    lam0 = np.repeat([-1.5, 0.0, 1.5], 4)
    M = Q @ np.diag(lam0) @ Q.T
    lam, T = O.jacobi_eigh(M)
    f = lambda x: np.exp(0.3j * x)
    ref = Q @ np.diag(f(lam0)) @ Q.T
    assert np.abs(T @ np.diag(f(lam)) @ T.T - ref).max() < 1e-13


def test_qr_mgs2_weighted_and_illconditioned():
    rng = np.random.default_rng(2)
    N, r, w = 500, 8, 0.37
    A = rng.standard_normal((N, r)) @ np.diag(10.0 ** (-1.5 * np.arange(r)))   # cond ~ 3e10
    A[:, 3] += 1e3 * A[:, 0]
    st = {}
    Q, R = O.qr_mgs2(A, w, st)
    assert st == {}
    assert np.abs(w * Q.T @ Q - np.eye(r)).max() < 1e-13
    assert np.abs(Q @ R - A).max() < 1e-13 * np.abs(A).max()
    assert np.allclose(R, np.triu(R)) and (np.diag(R) > 0).all()
    # rank-deficient input triggers the counted fallback and still returns an orthonormal basis
    A[:, 5] = A[:, 1]
    Q, R = O.qr_mgs2(A, w, st)
    assert st["qr_fallbacks"] == 1 and R[5, 5] == 0.0
    assert np.abs(w * Q.T @ Q - np.eye(r)).max() < 1e-12
    assert np.abs(Q @ R - A).max() < 1e-12 * np.abs(A).max()


def test_phi_functions():
    th = np.concatenate([np.linspace(-40, 40, 1601), [0.0, 1e-9, -1e-5, 0.999999, 1.0, -1.0, 1.000001]])
    z = (1j * th).astype(np.clongdouble)
    zs = np.where(th == 0, 1.0, z)
    # independent evaluation: long-double power series for |z| < 2, direct formula otherwise
    def series(shift):
        out = np.zeros(z.shape, dtype=np.clongdouble)
        term = np.full(z.shape, 1.0 / math.factorial(shift), dtype=np.clongdouble)
        for m in range(80):
            out = out + term
            term = term * z / (m + 1 + shift)
        return out
    p1 = np.where(np.abs(th) < 2, series(1), (np.exp(zs) - 1) / zs)
    p2 = np.where(np.abs(th) < 2, series(2), (np.exp(zs) - 1 - zs) / (zs * zs))
    assert np.abs(O.phi1_imag(th) - p1).max() < 4e-16
    assert np.abs(O.phi2_imag(th) - p2).max() < 4e-16
    assert O.phi1_imag(0.0) == 1.0 and O.phi2_imag(0.0) == 0.5


# ---------------- P3: closed forms at t = 0 ----------------
def test_initial_field_closed_form():
    """f0 of eq. (20): rho + 1 = -alpha sum cos(kappa x_i)  =>  E_i = -(alpha/kappa) sin(kappa x_i),
    electric energy 3/4 (alpha/kappa)^2 L^3, mass L^3 (up to the Maxwellian truncated at |v| = 6)."""
    cfg = inputs.make_config(2, n_x=16, n_v=32, r=3)
    gx, gv = grids(cfg)
    X, S, V = inputs.initial_factors(cfg)
    C1, C2, rho_t = O.coeff_C(V, gv)
    E = O.field(X @ S, rho_t, gx)
    a, k, L = cfg["alpha"], cfg["kappa"], cfg["x_hi"] - cfg["x_lo"]
    for d in range(3):
        assert np.abs(E[d] + (a / k) * np.sin(k * gx.coord_flat(d))).max() < 1e-9
    mom = O.moments(X, S, V, gx, gv)
    assert mom["electric_energy"] == pytest.approx(0.75 * (a / k) ** 2 * L ** 3, rel=1e-7)
    assert mom["electric_energy"] == pytest.approx(0.595320512, rel=1e-7)        # SURVEY P3, cfg 2
    assert mom["mass"] == pytest.approx(L ** 3, rel=1e-7)
    assert mom["kinetic_energy"] == pytest.approx(1.5 * L ** 3, rel=1e-6)         # 1/2 <|v|^2> = 3/2
    assert np.abs(mom["momentum"]).max() < 1e-7 * L ** 3        # left-closed grid keeps v=-6 only
    # f at probes reproduces the analytic f0
    ix, iv = inputs.probe_indices(cfg)
    xs = np.stack([gx.coord_flat(d)[ix] for d in range(3)])
    vs = np.stack([gv.coord_flat(d)[iv] for d in range(3)])
    f0 = (1 + a * np.cos(k * xs).sum(0)) * np.exp(-0.5 * (vs ** 2).sum(0)) / (2 * math.pi) ** 1.5
    assert np.abs(O.f_at(X, S, V, ix, iv) - f0).max() < 1e-14


def test_twostream_initial_energy():
    cfg = inputs.make_config(3, n_x=16, n_v=32, r=2)
    gx, gv = grids(cfg)
    X, S, V = inputs.initial_factors(cfg)
    mom = O.moments(X, S, V, gx, gv)
    assert mom["electric_energy"] == pytest.approx(0.581367688, rel=1e-6)        # 3/4 (1e-3/0.2)^2 (10 pi)^3
    assert mom["electric_energy"] == pytest.approx(0.75 * (1e-3 / 0.2) ** 2 * (10 * math.pi) ** 3, rel=1e-6)


# ---------------- P4: structure of the coefficients, exact free streaming ----------------
def test_coefficient_symmetries():
    cfg = inputs.make_config(1, n=8, r=6)
    gx, gv = grids(cfg)
    X, S, V = inputs.initial_factors(cfg)
    C1, C2, rho_t = O.coeff_C(V, gv)
    E = O.field(X @ S, rho_t, gx)
    D1, D2 = O.coeff_D(X, E, gx)
    for d in range(3):
        assert np.abs(C1[d] - C1[d].T).max() < 1e-14 and np.abs(D1[d] - D1[d].T).max() < 1e-14
        assert np.abs(C2[d] + C2[d].T).max() < 1e-14 and np.abs(D2[d] + D2[d].T).max() < 1e-14
    # definition written out with explicit loops on one entry (A^T diag(w) B)
    Vg = V.reshape(8, 8, 8, 6, order="F")                    # [i1, i2, i3, col]
    acc = 0.0
    for i1 in range(8):
        for i2 in range(8):
            for i3 in range(8):
                acc += gv.w * (cfg["v_lo"] + gv.h[1] * i2) * Vg[i1, i2, i3, 2] * Vg[i1, i2, i3, 4]
    assert C1[1][2, 4] == pytest.approx(acc, abs=1e-13)


def test_full_rank_C1_eigenvalues_are_grid_velocities():
    cfg = inputs.make_config(1, n=4, r=64, seed=11)
    gx, gv = grids(cfg)
    X, S, V = inputs.full_rank_factors(cfg, np.ones((64, 64)))
    C1, C2, _ = O.coeff_C(V, gv)
    for d in range(3):
        lam, _T = O.jacobi_eigh(C1[d].T)
        assert np.abs(np.sort(lam) - np.sort(gv.coord_flat(d))).max() < 1e-12


def test_K_flow_without_field_is_exact_free_streaming():
    """eqs. (17),(18) 'can be solved exactly in time': with E = 0 and V spanning the whole
    velocity grid the K-flow of ANY length t gives f0(x - v t, v), for Lie and Strang composition alike."""
    cfg = inputs.make_config(1, n_x=8, n_v=4, r=64, alpha=0.3, seed=12)
    gx, gv = grids(cfg)
    a, k = cfg["alpha"], cfg["kappa"]
    xs = [gx.coord_flat(d) for d in range(3)]
    vs = [gv.coord_flat(d) for d in range(3)]

    def f_exact(t):
        g = 1 + a * sum(np.cos(k * (xs[d][:, None] - vs[d][None, :] * t)) for d in range(3))
        return g * (np.exp(-0.5 * sum(v * v for v in vs)) / (2 * math.pi) ** 1.5)[None, :]
    rng = np.random.default_rng(12)
    Q, _ = np.linalg.qr(rng.standard_normal((64, 64)))
    V = Q / math.sqrt(gv.w)
    K0 = gv.w * f_exact(0.0) @ V
    C1, C2, _ = O.coeff_C(V, gv)
    E0 = np.zeros((3, gx.N))
    for t in (1.7, 13.0):
        for order in (1, 2):
            K = O.K_flow(K0, t, C1, C2, E0, gx, order)
            assert np.abs(K @ V.T - f_exact(t)).max() < 1e-12
            assert abs(np.sum(K * K) - np.sum(K0 * K0)) < 1e-12 * np.sum(K0 * K0)     # unitary

"""Seeded synthetic inputs shared by the oracle tests, the CUDA parity tests and bench.py.

Holds NONE of the method's arithmetic: only the grids/initial values of BASELINE.json's configs
(the paper's analytic initial conditions, eq. (20) PAPER.md:449-452 and the symmetric two-stream
variant of BASELINE.json config 3) turned into rank-r factors (X0, S0, V0), plus seeded probe
index pairs.  Imports numpy only (neither oracle/ nor the CUDA binding).

Factors: (N, r) float64 arrays in Fortran order (= the C ABI's column-major layout), row index
I = i1 + n1*(i2 + n2*i3);  h^3 X^T X = I,  h^3 V^T V = I;  f0 = X0 S0 V0^T.
"""
import math
import numpy as np

TWO_PI = 2.0 * math.pi

CONFIGS = {
    # name: n, r, x-domain, v-domain, problem, alpha, kappa, tau, steps
    1: dict(n=8, r=5, x_lo=0.0, x_hi=4 * math.pi, v_lo=-6.0, v_hi=6.0, problem="landau",
            alpha=0.01, kappa=0.5, tau=0.1, steps=20),
    2: dict(n=32, r=10, x_lo=0.0, x_hi=4 * math.pi, v_lo=-6.0, v_hi=6.0, problem="landau",
            alpha=0.01, kappa=0.5, tau=0.1, steps=200),
    3: dict(n=64, r=10, x_lo=0.0, x_hi=10 * math.pi, v_lo=-9.0, v_hi=9.0, problem="twostream",
            alpha=1e-3, kappa=0.2, v0=2.4, tau=0.05, steps=100),
    4: dict(n=128, r=15, x_lo=0.0, x_hi=4 * math.pi, v_lo=-6.0, v_hi=6.0, problem="landau",
            alpha=0.5, kappa=0.5, tau=0.05, steps=50),
    5: dict(n=256, r=20, x_lo=0.0, x_hi=4 * math.pi, v_lo=-6.0, v_hi=6.0, problem="landau",
            alpha=0.01, kappa=0.5, tau=0.05, steps=10, rank20_amp=1e-6, band=4),
    # not a BASELINE.json config: the paper's own two-stream initial value, eq. (21), the workload of
    # its Table 4 and Section 6.3: v_bar = (5/2, 0, 0), v_tilde = (-5/2, -9/4, -2), norm 1/sqrt((8 pi)^3)
    6: dict(n=64, r=10, x_lo=0.0, x_hi=10 * math.pi, v_lo=-9.0, v_hi=9.0, problem="twostream_paper",
            alpha=1e-3, kappa=0.2, v_bar=(2.5, 0.0, 0.0), v_til=(-2.5, -2.25, -2.0), tau=0.01, steps=100),
}


def make_config(idx=None, **over):
    """dict describing one workload; idx in 1..5 = BASELINE.json configs[idx-1]; keyword overrides
    (n, n_x, n_v, r, tau, steps, alpha, ...) give the scaled-down variants used by the tests."""
    c = dict(CONFIGS[idx]) if idx is not None else dict(CONFIGS[1])
    c.update(over)
    c.setdefault("n_x", c["n"])
    c.setdefault("n_v", c["n"])
    c["seed"] = c.get("seed", 1000 + (idx or 0))
    return c


def grid_axes(n, lo, hi):
    """coordinates of the left-closed periodic grid, per dimension"""
    h = (hi - lo) / n
    return lo + h * np.arange(n), h


def _outer3(a1, a2, a3):
    """flattened (I = i1 + n1*(i2 + n2*i3)) tensor product a1(x1) a2(x2) a3(x3)"""
    return (a3[:, None, None] * a2[None, :, None] * a1[None, None, :]).reshape(-1)


def _sum3(a1, a2, a3):
    return (a3[:, None, None] + a2[None, :, None] + a1[None, None, :]).reshape(-1)


def _band_limited_columns(rng, n, ncols, band):
    """seeded real random columns whose Fourier content is limited to |m_d| <= band"""
    cols = np.empty((n ** 3, ncols), order="F")
    nb = 2 * band + 1
    for c in range(ncols):
        spec = np.zeros((n, n, n // 2 + 1), dtype=complex)
        co = rng.standard_normal((nb, nb, band + 1)) + 1j * rng.standard_normal((nb, nb, band + 1))
        idx = np.r_[0:band + 1, n - band:n]
        spec[np.ix_(idx, idx, np.arange(band + 1))] = co
        cols[:, c] = np.fft.irfftn(spec, s=(n, n, n), axes=(0, 1, 2)).reshape(-1)
    return cols


def _orthonormal_factor(first, pad, h3):
    """[first | pad] -> weighted-orthonormal basis whose first column is first/||first||_w"""
    A = np.column_stack([first, pad]) if pad.shape[1] else first[:, None]
    Q, R = np.linalg.qr(A)
    sg = np.sign(np.diag(R))
    sg[sg == 0] = 1.0
    Q = Q * sg[None, :]
    return np.asfortranarray(Q / math.sqrt(h3)), abs(R[0, 0]) * math.sqrt(h3)


def initial_factors(cfg):
    """(X0, S0, V0) of the separable initial value f0 = g(x) M(v), rank 1 padded to rank r with seeded
    random orthonormal columns (zero weight in S0, configs 1-4) or band-limited columns carrying weight
    rank20_amp (config 5)."""
    nx, nv, r = cfg["n_x"], cfg["n_v"], cfg["r"]
    x, hx = grid_axes(nx, cfg["x_lo"], cfg["x_hi"])
    v, hv = grid_axes(nv, cfg["v_lo"], cfg["v_hi"])
    a, k = cfg["alpha"], cfg["kappa"]
    g = 1.0 + a * _sum3(np.cos(k * x), np.cos(k * x), np.cos(k * x))
    m1 = np.exp(-0.5 * v * v) / math.sqrt(TWO_PI)
    if cfg["problem"] == "landau":
        M = _outer3(m1, m1, m1)
    elif cfg["problem"] == "twostream":
        v0 = cfg["v0"]
        b1 = 0.5 * (np.exp(-0.5 * (v - v0) ** 2) + np.exp(-0.5 * (v + v0) ** 2)) / math.sqrt(TWO_PI)
        M = _outer3(b1, m1, m1)
    elif cfg["problem"] == "twostream_paper":
        b = [(np.exp(-0.5 * (v - vb) ** 2) + np.exp(-0.5 * (v - vt) ** 2)) / math.sqrt(4.0 * TWO_PI)
             for vb, vt in zip(cfg["v_bar"], cfg["v_til"])]
        M = _outer3(b[0], b[1], b[2])
    else:
        raise ValueError(cfg["problem"])
    rng = np.random.default_rng(cfg["seed"])
    band = cfg.get("band")
    if band is None:
        padx = rng.standard_normal((nx ** 3, r - 1))
        padv = rng.standard_normal((nv ** 3, r - 1))
    else:
        padx = _band_limited_columns(rng, nx, r - 1, band)
        padv = _band_limited_columns(rng, nv, r - 1, band)
    X0, ngx = _orthonormal_factor(g, padx, hx ** 3)
    V0, nMv = _orthonormal_factor(M, padv, hv ** 3)
    S0 = np.zeros((r, r), order="F")
    S0[0, 0] = ngx * nMv
    amp = cfg.get("rank20_amp")
    if amp:
        for j in range(1, r):
            S0[j, j] = amp * S0[0, 0]
    return X0, S0, V0


def full_rank_factors(cfg, F):
    """for the n=4 full-rank checks: factors (X, S, V) with r = N of an arbitrary (N_x, N_v) matrix F,
    X S V^T = F.  X, V are seeded random orthonormal bases (not the SVD basis), S = h^6 X^T F V."""
    nx, nv = cfg["n_x"], cfg["n_v"]
    hx = (cfg["x_hi"] - cfg["x_lo"]) / nx
    hv = (cfg["v_hi"] - cfg["v_lo"]) / nv
    rng = np.random.default_rng(cfg["seed"])
    Qx, _ = np.linalg.qr(rng.standard_normal((nx ** 3, nx ** 3)))
    Qv, _ = np.linalg.qr(rng.standard_normal((nv ** 3, nv ** 3)))
    X = np.asfortranarray(Qx / math.sqrt(hx ** 3))
    V = np.asfortranarray(Qv / math.sqrt(hv ** 3))
    S = np.asfortranarray((hx ** 3 * hv ** 3) * (X.T @ F @ V))
    return X, S, V


def f0_full(cfg):
    """the full (N_x, N_v) matrix of f0 (tiny grids only)"""
    X0, S0, V0 = initial_factors(dict(cfg, r=1))
    return (X0 * S0[0, 0]) @ V0.T


def probe_indices(cfg, nprobe=64, seed=7):
    """seeded probe index pairs (ix, iv), uniform in [0, N_x) x [0, N_v)"""
    rng = np.random.default_rng(seed)
    ix = rng.integers(0, cfg["n_x"] ** 3, size=nprobe).astype(np.int64)
    iv = rng.integers(0, cfg["n_v"] ** 3, size=nprobe).astype(np.int64)
    return ix, iv


def weighted_start(cfg, decay=1e-2, seed=77):
    """(X0, S0, V0) of initial_factors(cfg) with a FULL-RANK coupling matrix: S0 = U diag(s) W^T, s from sigma_1 down to
    decay * sigma_1 (geometric), U, W seeded orthogonal matrices that leave the physical first column alone.  Every basis
    direction then carries weight, so the bases an integrator computes from K = X S, L = V S^T are determined to rounding
    (needed where the result depends on them, e.g. the unconventional integrator: tests/test_gpu_parity.py)."""
    X, S, V = initial_factors(cfg)
    r = cfg["r"]
    rng = np.random.default_rng(seed)
    mats = []
    for _ in range(2):
        A = rng.standard_normal((r, r))
        A[0, :] = 0.0
        A[:, 0] = 0.0
        A[0, 0] = 1.0
        Q, _ = np.linalg.qr(A)
        mats.append(Q)
    s = S[0, 0] * np.logspace(0.0, np.log10(decay), r)
    return X, mats[0] @ np.diag(s) @ mats[1].T, V


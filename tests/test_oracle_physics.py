"""P7-P10: order of convergence of the oracle's Algorithms 1 and 2 (paper section 6.1
protocol scaled down), the linear Landau damping rate, free streaming through the full step, invariants."""
import math

import numpy as np
import pytest

from oracle import dlr_oracle as O
from paper_2110_13481_b200 import inputs


def grids(cfg):
    gx = O.Grid3((cfg["n_x"],) * 3, (cfg["x_lo"],) * 3, (cfg["x_hi"],) * 3)
    gv = O.Grid3((cfg["n_v"],) * 3, (cfg["v_lo"],) * 3, (cfg["v_hi"],) * 3)
    return gx, gv


@pytest.mark.slow
def test_orders_of_convergence():
    """Fig. 3: Algorithm 1 converges with order 1, Algorithm 2 with order 2.
    n = 8, r = 10 (r >= 7 so that the limit is unique), T = 1; successive differences
    |f_m - f_2m| must shrink by 2 (Alg. 1) and 4 (Alg. 2).  A wrong E^{1/2} predictor or a first-order
    third sub-flow inside Algorithm 2 shows up as a ratio of 2."""
    cfg = inputs.make_config(1, n=8, r=10)
    gx, gv = grids(cfg)
    X0, S0, V0 = inputs.initial_factors(cfg)

    def run(m, step):
        X, S, V = X0, S0, V0
        for _ in range(m):
            X, S, V = step(X, S, V, 1.0 / m, gx, gv)
        return X @ S @ V.T
    f2 = [run(m, O.step_alg2) for m in (8, 16, 32, 64)]
    d2 = [np.abs(f2[i] - f2[i + 1]).max() for i in range(3)]
    assert 3.3 < d2[0] / d2[1] < 5.0 and 3.3 < d2[1] / d2[2] < 5.0
    f1 = [run(m, O.step_alg1) for m in (8, 16, 32)]
    d1 = [np.abs(f1[i] - f1[i + 1]).max() for i in range(2)]
    assert 1.8 < d1[0] / d1[1] < 2.25
    # both algorithms approach the same limit, Algorithm 2 much faster
    assert np.abs(f1[2] - f2[3]).max() < 3 * d1[1]
    assert d2[2] < 0.02 * d1[1]


@pytest.mark.slow
def test_linear_landau_damping_rate():
    """Linear Landau damping, k = 0.5: the electric energy decays at 'the expected theoretical exponential
    rate', gamma = -0.1533 and omega = 1.4156 from linear theory (BASELINE.json).
    Grid 8^3 x 16^3 (one resolved mode per direction in x), r = 10, tau = 0.1, T = 9.6."""
    cfg = inputs.make_config(2, n_x=8, n_v=16, r=10)
    gx, gv = grids(cfg)
    X, S, V = inputs.initial_factors(cfg)
    tau = 0.1
    X, S, V, hist, _, stats = O.run(X, S, V, tau, 96, gx, gv)
    assert stats == {}
    ee = np.array([h["electric_energy"] for h in hist])
    mass = np.array([h["mass"] for h in hist])
    assert np.abs(mass / mass[0] - 1).max() < 1e-7              # paper: ~3e-8 (not exactly conserved)
    tp, lp = [], []
    for i in range(1, len(ee) - 1):
        if ee[i] > ee[i - 1] and ee[i] > ee[i + 1]:
            y0, y1, y2 = np.log(ee[i - 1:i + 2])
            d = 0.5 * (y0 - y2) / (y0 - 2 * y1 + y2)
            tp.append(tau * (i + d))
            lp.append(y1 - 0.25 * (y0 - y2) * d)
    assert len(tp) == 4
    gamma = 0.5 * np.polyfit(tp, lp, 1)[0]
    assert gamma == pytest.approx(-0.1533, rel=0.03)
    assert np.diff(tp).mean() == pytest.approx(math.pi / 1.4156, rel=0.01)


def test_full_step_without_field_converges_to_free_streaming():
    """E = 0 (e_scale = 0): the exact solution is f0(x - v t, v), of rank 1 + 2*3 = 7.  The full step is not
    exact (the L-flow treats -v.L.D2^T explicitly) but must converge to it at second order (r = 8)."""
    cfg = inputs.make_config(1, n=8, r=8, alpha=0.2)
    gx, gv = grids(cfg)
    X0, S0, V0 = inputs.initial_factors(cfg)
    a, k = cfg["alpha"], cfg["kappa"]
    xs = [gx.coord_flat(d) for d in range(3)]
    vs = [gv.coord_flat(d) for d in range(3)]
    T = 0.5
    g = 1 + a * sum(np.cos(k * (xs[d][:, None] - vs[d][None, :] * T)) for d in range(3))
    exact = g * (np.exp(-0.5 * sum(v * v for v in vs)) / (2 * math.pi) ** 1.5)[None, :]
    errs = []
    for m in (4, 8, 16):
        X, S, V = X0, S0, V0
        for _ in range(m):
            X, S, V = O.step_alg2(X, S, V, T / m, gx, gv, e_scale=0.0)
        errs.append(np.abs(X @ S @ V.T - exact).max())
    assert 3.5 < errs[0] / errs[1] < 4.5 and 3.5 < errs[1] / errs[2] < 4.5
    assert errs[2] < 1e-4 * np.abs(exact).max()


def test_invariants_config1():
    """cfg 1 (parity-only config): ||S||_F drifts only slowly, no QR fallback, factors stay orthonormal."""
    cfg = inputs.make_config(1)
    gx, gv = grids(cfg)
    X, S, V = inputs.initial_factors(cfg)
    assert math.sqrt(np.sum(S * S)) == pytest.approx(6.925561965855, rel=1e-12)    # = ||f0||_{L2}, analytic part
    X, S, V, hist, _, stats = O.run(X, S, V, cfg["tau"], 5, gx, gv)
    assert stats == {}
    assert abs(hist[-1]["s_fro"] / hist[0]["s_fro"] - 1) < 1e-6
    assert np.abs(gx.w * X.T @ X - np.eye(5)).max() < 1e-13 and np.abs(gv.w * V.T @ V - np.eye(5)).max() < 1e-13
    assert hist[0]["electric_energy"] == pytest.approx(0.59642764081, rel=1e-10)   # 8-point quadrature value

"""P5/P6: the oracle's whole low-rank algebra against brute-force full-grid solvers
at n = 4 (tests/bruteforce6d.py, written independently of oracle/).  CPU only."""
import numpy as np
import pytest

from oracle import dlr_oracle as O
from paper_2110_13481_b200 import inputs
from bruteforce6d import Mirrored


def _setup(seed=5):
    cfg = inputs.make_config(1, n=4, r=64, alpha=0.05, v_lo=-3.0, v_hi=3.0, seed=seed)
    F0 = inputs.f0_full(cfg)
    F0 = F0 * (1 + 0.2 * np.random.default_rng(3).standard_normal(F0.shape))      # generic full-rank data
    gx = O.Grid3((4,) * 3, (cfg["x_lo"],) * 3, (cfg["x_hi"],) * 3)
    gv = O.Grid3((4,) * 3, (cfg["v_lo"],) * 3, (cfg["v_hi"],) * 3)
    bf = Mirrored(4, cfg["x_lo"], cfg["x_hi"], cfg["v_lo"], cfg["v_hi"])
    return cfg, F0, gx, gv, bf


@pytest.mark.slow
def test_full_rank_dlr_equals_mirrored_bruteforce():
    """At r = N_x = N_v the projectors are the identity, so Algorithm 2 on the factors and the same
    sequence of flows on the full 6D array are the same map: agreement to rounding over 2 steps, for
    Algorithm 1 and Algorithm 2; mass is conserved to rounding (it is only at full rank)."""
    cfg, F0, gx, gv, bf = _setup()
    X, S, V = inputs.full_rank_factors(cfg, F0)
    assert np.abs(X @ S @ V.T - F0).max() < 1e-14
    F = F0.reshape((4,) * 6).copy()
    tau = 0.1
    m0 = O.moments(X, S, V, gx, gv)
    assert m0["mass"] == pytest.approx(bf.mass(F), rel=1e-13)
    assert m0["electric_energy"] == pytest.approx(bf.electric_energy(F), rel=1e-12)
    for _ in range(2):
        X, S, V = O.step_alg2(X, S, V, tau, gx, gv)
        F = bf.step_alg2(F, tau)
        Fd = (X @ S @ V.T).reshape((4,) * 6)
        assert np.abs(Fd - F).max() <= 2e-12 * np.abs(F).max()
        mom = O.moments(X, S, V, gx, gv)
        assert mom["mass"] == pytest.approx(m0["mass"], rel=2e-12)
        assert mom["electric_energy"] == pytest.approx(bf.electric_energy(F), rel=1e-10)
    assert np.abs(F - F0.reshape((4,) * 6)).max() > 1e-2 * np.abs(F0).max()        # something happened
    # Algorithm 1 (one step, from the evolved state)
    X1, S1, V1 = O.step_alg1(X, S, V, tau, gx, gv)
    F1 = bf.step_alg1(F, tau)
    assert np.abs((X1 @ S1 @ V1.T).reshape((4,) * 6) - F1).max() <= 2e-12 * np.abs(F1).max()


def test_mirrored_scheme_converges_at_second_order_to_classical_strang():
    """The sequence of flows of Algorithm 2 (predictor for E^{1/2}, Strang K-S-L-S-K, ETD2RK third
    sub-flows) is a second-order integrator of the Vlasov-Poisson system: its distance to an independent
    classical Strang splitting falls like tau^2 (ratio -> 4); Algorithm 1's falls like tau (ratio -> 2).
    Together with the test above this pins the oracle's scheme (R8, R10, R13) to 'solves eq. (1) at order 2'."""
    cfg, F0, gx, gv, bf = _setup()
    F0 = F0.reshape((4,) * 6)
    T = 0.4

    def run(stepper, m):
        F = F0.copy()
        for _ in range(m):
            F = stepper(F, T / m)
        return F
    ref = run(bf.classical_strang, 512)
    e2 = [np.abs(run(bf.step_alg2, m) - ref).max() for m in (8, 16, 32)]
    e1 = [np.abs(run(bf.step_alg1, m) - ref).max() for m in (8, 16, 32)]
    assert 3.6 < e2[0] / e2[1] < 4.4 and 3.8 < e2[1] / e2[2] < 4.2
    assert 1.8 < e1[0] / e1[1] < 2.2 and 1.9 < e1[1] / e1[2] < 2.1
    assert e2[2] < 0.05 * e1[2]

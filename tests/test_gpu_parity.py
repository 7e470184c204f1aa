"""GPU parity: the CUDA path (through the C ABI, paper_2110_13481_b200.dlr) against the oracle on the same seeded
inputs, compared on gauge-invariant quantities only (QR sign/rotation and eigenvector choice are free):
f at 64 seeded probe pairs normalised by max_p |f|, electric energy, mass.
Tolerance (BASELINE.json north_star): relative error <= 1e-10 after one step, <= 1e-8 after the full run."""
import json
import math
import os

import numpy as np
import pytest

from oracle import dlr_oracle as O
from paper_2110_13481_b200 import inputs

pytestmark = pytest.mark.gpu
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
TOL_STEP, TOL_RUN = 1e-10, 1e-8


def grids(cfg):
    gx = O.Grid3((cfg["n_x"],) * 3, (cfg["x_lo"],) * 3, (cfg["x_hi"],) * 3)
    gv = O.Grid3((cfg["n_v"],) * 3, (cfg["v_lo"],) * 3, (cfg["v_hi"],) * 3)
    return gx, gv


def rel(a, b):
    return abs(a - b) / abs(b)


def ee_scale(hist, m):
    """normalisation of the electric-energy error at step m of a history (reading R17): the value itself,
    except at a strict local minimum of the oracle's history, where the field passes (almost) through zero and the
    pointwise relative error of 1/2 |E|^2 is ill-conditioned (fp64 rounding floor ~1e-13 * ee(0) divided by a value
    1e-5 * ee(0)); there the larger of the two neighbouring samples is used."""
    if 0 < m < len(hist) - 1 and hist[m] < hist[m - 1] and hist[m] < hist[m + 1]:
        return max(hist[m - 1], hist[m + 1])
    return hist[m]


def make_ctx(cfg, order=2, e_scale=1.0, flags=0):
    from paper_2110_13481_b200 import dlr
    return dlr.Dlr(dlr.config_from_inputs(cfg, order=order, e_scale=e_scale, flags=flags))


def check(ctx, Xo, So, Vo, gx, gv, ix, iv, tol, e_scale=1.0):
    m, f = ctx.moments(ix, iv)
    mo = O.moments(Xo, So, Vo, gx, gv, e_scale)
    fo = O.f_at(Xo, So, Vo, ix, iv)
    assert m["qr_fallbacks"] == 0 and m["nonfinite"] == 0 and m["eig_unconverged"] == 0
    assert np.abs(f - fo).max() <= tol * np.abs(fo).max()
    assert rel(m["mass"], mo["mass"]) <= tol
    if e_scale:
        assert rel(m["electric_energy"], mo["electric_energy"]) <= tol
    assert rel(m["kinetic_energy"], mo["kinetic_energy"]) <= tol
    assert rel(m["s_fro"], mo["s_fro"]) <= tol
    for d in range(3):
        assert abs(m["momentum"][d] - mo["momentum"][d]) <= tol * mo["mass"]


@pytest.mark.parametrize("n,r", [(8, 5), (16, 10), (32, 10), (16, 8), (16, 15), (16, 20)])
def test_fft_against_numpy(n, r):
    """the hand-written batched 3D r2c/c2r FFT of the Poisson solve (three shared-memory passes, 3 columns) against
    numpy.fft; the spectrum is compared in the library's layout (k1 natural 0..n/2, k2/k3 at bit-reversed
    positions).  The 1D transforms inside the K/L-flow passes are covered by the step parity tests below."""
    cfg = inputs.make_config(1, n=n, r=r)
    ctx = make_ctx(cfg)
    rng = np.random.default_rng(n + r)
    lg = int(math.log2(n))
    br = np.array([int(format(i, f"0{lg}b")[::-1], 2) for i in range(n)])
    for ncols in (3,):
        A = np.asfortranarray(rng.standard_normal((n ** 3, ncols)))
        back, spec = ctx.test_fft_roundtrip(0, A)
        ref = np.fft.rfftn(A.T.reshape(ncols, n, n, n), axes=(1, 2, 3))[:, br][:, :, br]
        assert np.abs(back - A).max() < 1e-13
        assert np.abs(spec - ref).max() < 1e-13 * np.abs(ref).max()
    ctx.close()


@pytest.mark.parametrize("n,r,order,e_scale", [
    (8, 5, 2, 1.0), (8, 5, 1, 1.0), (8, 5, 2, 0.0), (16, 10, 2, 1.0), (16, 10, 1, 1.0), (32, 10, 2, 1.0),
    (16, 8, 2, 1.0), (16, 15, 2, 1.0), (16, 20, 2, 1.0)])
def test_one_and_two_steps_match_oracle(n, r, order, e_scale):
    """one step (first step: direct launches, computes C(V0)) and a second step (CUDA-graph replay, reuses the C
    coefficients of V1) against the oracle; n = 16, 32 span several tiles with ragged tails (n/2+1 odd)."""
    cfg = inputs.make_config(1, n=n, r=r)
    gx, gv = grids(cfg)
    X, S, V = inputs.initial_factors(cfg)
    ix, iv = inputs.probe_indices(cfg)
    ctx = make_ctx(cfg, order, e_scale)
    ctx.set_initial(X, S, V)
    check(ctx, X, S, V, gx, gv, ix, iv, 1e-13, e_scale)
    step = O.step_alg2 if order == 2 else O.step_alg1
    for _ in range(2):
        ctx.step(cfg["tau"])
        X, S, V = step(X, S, V, cfg["tau"], gx, gv, e_scale)
        check(ctx, X, S, V, gx, gv, ix, iv, TOL_STEP, e_scale)
    Xg, Sg, Vg = ctx.get_factors()
    assert np.abs(gx.w * Xg.T @ Xg - np.eye(r)).max() < 1e-12
    assert np.abs(gv.w * Vg.T @ Vg - np.eye(r)).max() < 1e-12
    ctx.close()


@pytest.mark.parametrize("n_x,n_v,r", [(8, 8, 5), (16, 16, 10), (16, 16, 15), (16, 16, 20), (32, 16, 8), (16, 32, 10), (64, 64, 10)])
@pytest.mark.parametrize("start", ["full_rank", "rank_one"])
def test_unconventional_integrator_matches_oracle(n_x, n_v, r, start):
    """DLR_FLAG_UNCONVENTIONAL (the integrator of the paper's reference [4], named in PAPER.md:29, 288) against
    oracle.step_bug: three steps (direct launches, graph capture, graph replay) compared on f at the probes, mass,
    energies, momentum, ||S||_F.
    full_rank: S0 with singular values sigma_1 ... 1e-2 sigma_1 (inputs.weighted_start): north_star's one-step tolerance
      1e-10 at every step.
    rank_one: config 1 as it is (S0 of rank 1).  There several columns of K1, L1 are rounding noise, the QR completes the
      bases with rounding-determined directions, and - unlike the projector-splitting integrators - the Galerkin S step
      evolves in them: the ORACLE ITSELF, with K1 and L1 perturbed by 1e-16 relative before the QR, moves by 1.6e-10 in f and
      8.8e-10 in the electric energy after one step at 16^3, r = 10 (Algorithm 1: 6e-13; with the full-rank start: 1e-14;
      DESIGN.md reading R19), and the amplification grows with the grid (GPU vs oracle at 64^3: 4e-8).  Several results are
      equally correct there, so this case checks what is valid for all of them - no QR repair, nothing non-finite,
      orthonormal bases - and agreement to 1e-6, a sanity bound on the rounding-level ambiguity, not a parity claim."""
    from paper_2110_13481_b200 import dlr
    cfg = inputs.make_config(1, n_x=n_x, n_v=n_v, r=r)
    gx, gv = grids(cfg)
    X, S, V = inputs.weighted_start(cfg) if start == "full_rank" else inputs.initial_factors(cfg)
    tol = TOL_STEP if start == "full_rank" else 1e-6
    ix, iv = inputs.probe_indices(cfg)
    ctx = make_ctx(cfg, order=1, flags=dlr.FLAG_UNCONVENTIONAL)
    ctx.set_initial(X, S, V)
    for _ in range(3):
        ctx.step(cfg["tau"])
        X, S, V = O.step_bug(X, S, V, cfg["tau"], gx, gv)
        check(ctx, X, S, V, gx, gv, ix, iv, tol)
    Xg, Sg, Vg = ctx.get_factors()
    assert np.abs(gx.w * Xg.T @ Xg - np.eye(r)).max() < 1e-12
    assert np.abs(gv.w * Vg.T @ Vg - np.eye(r)).max() < 1e-12
    ctx.close()
    # the flag needs order = 1
    with pytest.raises(dlr.DlrError):
        make_ctx(cfg, order=2, flags=dlr.FLAG_UNCONVENTIONAL)


def test_anisotropic_grid_and_half_step_field():
    """n_x != n_v (the paper's headline shapes are anisotropic) and the field E^{1/2} of Algorithm 2
    line 2 itself, compared point-wise."""
    cfg = inputs.make_config(2, n_x=8, n_v=16, r=10)
    gx, gv = grids(cfg)
    X, S, V = inputs.initial_factors(cfg)
    ix, iv = inputs.probe_indices(cfg)
    ctx = make_ctx(cfg)
    ctx.set_initial(X, S, V)
    ctx.step(0.1)
    X1, L1, _ = O.step_alg1(X, S, V, 0.05, gx, gv, upto9=True)
    Ehalf = O.field(X1, L1.T @ (gv.w * np.ones(gv.N)), gx)
    assert np.abs(ctx.get_field() - Ehalf).max() <= 1e-11 * np.abs(Ehalf).max()
    X, S, V = O.step_alg2(X, S, V, 0.1, gx, gv)
    check(ctx, X, S, V, gx, gv, ix, iv, TOL_STEP)
    ctx.close()


def test_full_run_config1():
    """BASELINE.json config 1 (8^3 x 8^3, r = 5, tau = 0.1, 20 steps): electric energy per step and f at the 64
    probes, against the oracle run live."""
    cfg = inputs.make_config(1)
    gx, gv = grids(cfg)
    X, S, V = inputs.initial_factors(cfg)
    ix, iv = inputs.probe_indices(cfg)
    ctx = make_ctx(cfg)
    ctx.set_initial(X, S, V)
    ee_gpu, ee_ora = [ctx.moments()["electric_energy"]], [O.moments(X, S, V, gx, gv)["electric_energy"]]
    for _ in range(cfg["steps"]):
        ctx.step(cfg["tau"])
        X, S, V = O.step_alg2(X, S, V, cfg["tau"], gx, gv)
        ee_gpu.append(ctx.moments()["electric_energy"])
        ee_ora.append(O.moments(X, S, V, gx, gv)["electric_energy"])
    for m in range(len(ee_ora)):
        assert abs(ee_gpu[m] - ee_ora[m]) <= (TOL_STEP if m <= 1 else TOL_RUN) * ee_scale(ee_ora, m), m
    check(ctx, X, S, V, gx, gv, ix, iv, TOL_RUN)
    ctx.close()


def _golden_run(idx, max_steps=None, name=None, **over):
    """run the GPU path against a stored oracle run (tests/golden/, written by make_golden.py from oracle/ alone).
    Returns (golden, GPU electric-energy history)."""
    path = os.path.join(GOLDEN, name or f"cfg{idx}.json")
    if not os.path.exists(path):
        pytest.skip(f"{path} not generated")
    gold = json.load(open(path))
    cfg = inputs.make_config(idx, **over)
    X, S, V = inputs.initial_factors(cfg)
    ix, iv = inputs.probe_indices(cfg)
    ctx = make_ctx(cfg)
    ctx.set_initial(X, S, V)
    nsteps = gold["steps"] if max_steps is None else min(max_steps, gold["steps"])
    assert gold["qr_fallbacks"] == 0
    ee_gpu, worst_pt = [], 0.0
    for step in range(nsteps + 1):
        if step:
            ctx.step(cfg["tau"])
        tol = TOL_STEP if step <= 1 else TOL_RUN
        if str(step) in gold["f_probe"]:
            m, f = ctx.moments(ix, iv)
            fo = np.array(gold["f_probe"][str(step)])
            assert np.abs(f - fo).max() <= tol * np.abs(fo).max(), step
        else:
            m = ctx.moments()
        ee = gold["electric_energy"]
        ee_gpu.append(m["electric_energy"])
        worst_pt = max(worst_pt, rel(m["electric_energy"], ee[step]))
        assert abs(m["electric_energy"] - ee[step]) <= tol * ee_scale(ee[:nsteps + 1], step), step
        assert rel(m["mass"], gold["mass"][step]) <= tol, step
        assert rel(m["kinetic_energy"], gold["kinetic_energy"][step]) <= tol, step
        assert rel(m["s_fro"], gold["s_fro"][step]) <= tol, step
        assert m["qr_fallbacks"] == 0 and m["nonfinite"] == 0 and m["eig_unconverged"] == 0
    ctx.close()
    # the literal tolerance of north_star is pointwise; reading R17 normalises strict local minima by their
    # neighbours.  Both are reported; relative to max_t ee the history error is far below either.
    err_hist = np.abs(np.array(ee_gpu) - np.array(ee[:nsteps + 1])).max() / max(ee[:nsteps + 1])
    print(f"golden {os.path.basename(path)}: electric-energy history: worst pointwise rel. error {worst_pt:.2e}, "
          f"max |diff| / max ee {err_hist:.2e}")
    assert err_hist <= 0.1 * TOL_RUN
    return gold, np.array(ee_gpu)


def test_full_run_config2_golden_and_damping_rate():
    """BASELINE.json config 2 (32^3 x 32^3, r = 10, 200 steps) against tests/golden/cfg2.json (written by
    tests/golden/make_golden.py from the oracle); the GPU energy history shows the Landau rate -0.1533."""
    gold, ee = _golden_run(2)                   # ee: the GPU history (it matches the oracle's to 1e-8, checked above)
    tau = gold["tau"]
    tp, lp = [], []
    for i in range(1, len(ee) - 1):
        if ee[i] > ee[i - 1] and ee[i] > ee[i + 1] and tau * i < 16.5:
            tp.append(tau * i)
            lp.append(math.log(ee[i]))
    gamma = 0.5 * np.polyfit(tp, lp, 1)[0]
    assert gamma == pytest.approx(-0.1533, rel=0.04)


def test_config3_metric_shape_golden():
    """BASELINE.json config 3 = the metric's shape (64^3 x 64^3, r = 10, two-stream), in the launch configuration
    bench.py times, against tests/golden/cfg3.json for as many steps as the golden file holds."""
    _golden_run(3)


@pytest.mark.parametrize("base,n_x,n_v,r", [(5, 64, 64, 20), (4, 64, 64, 15), (5, 128, 128, 20), (2, 32, 128, 10),
                                            (4, 128, 32, 15)])
def test_one_step_at_every_tile_shape_live_oracle(base, n_x, n_v, r):
    """every (n, r) combination takes its own tile shape, CTA size and occupancy rule in the pass kernels
    (api.cu::setup_grid, kernels_dir.cuh launch bounds): one step of Algorithm 2 against the oracle run live at the
    shapes that the other tests do not reach: r = 20 and r = 15 at n = 64 (one CTA per SM at r = 20), r = 20 at
    n = 128 (single-line tiles holding all of the shared memory, three FFT groups), mixed 32/128 grids.
    Inputs: the recipe of BASELINE.json config `base` at these grids; r = 20 uses config 5's (band-limited rank-20
    perturbation at 1e-6): with the rank-1 initial value of configs 1-4 the first K at r = 20, n >= 64 is rank
    deficient to working precision, the oracle's QR replaces columns (reading R12) and the step is then defined only
    up to that choice (measured: E^{1/2} moves by 3e-6) - parity needs a fallback-free oracle step, asserted here."""
    cfg = inputs.make_config(base, n_x=n_x, n_v=n_v, r=r)
    gx, gv = grids(cfg)
    X, S, V = inputs.initial_factors(cfg)
    ix, iv = inputs.probe_indices(cfg)
    ctx = make_ctx(cfg)
    ctx.set_initial(X, S, V)
    ctx.step(cfg["tau"])
    stats = {}
    X, S, V = O.step_alg2(X, S, V, cfg["tau"], gx, gv, 1.0, stats)
    assert stats.get("qr_fallbacks", 0) == 0
    check(ctx, X, S, V, gx, gv, ix, iv, TOL_STEP)
    ctx.close()


@pytest.mark.parametrize("base,n_x,n_v,r", [(2, 256, 8, 10), (2, 8, 256, 10), (5, 16, 256, 20)])
def test_one_step_at_n256_golden(base, n_x, n_v, r):
    """the n = 256 kernel paths (three radix groups, single-line 227 KB tiles, and at r = 20 one CTA per SM with up to
    255 registers) on the x grid and on the v grid: one step against tests/golden/shape_<n_x>_<n_v>_<r>.json, an
    oracle step (10-20 minutes of host time each, hence stored) written by tests/golden/make_golden.py."""
    _golden_run(base, name=f"shape_{n_x}_{n_v}_{r}.json", n_x=n_x, n_v=n_v, r=r)


def test_config5_one_step_golden():
    """BASELINE.json config 5 (256^3 x 256^3, r = 20, band-limited rank-20 perturbation) at FULL size, in the launch
    configuration bench.py times: one step against tests/golden/cfg5.json (an oracle step needs ~35 GB and about an
    hour of host time, hence stored; written by tests/golden/make_golden.py 5 1)."""
    _golden_run(5)


def test_predictor_L_shortcut_equals_the_flow():
    """the predictor of Algorithm 2 takes rho(L^1) from the 1D marginals of V instead of running the L flow (DESIGN.md
    row a7').  A/B against the literal flow (DLR_FLAG_PREDICTOR_L_FLOW) after several steps, when S has full rank and
    the field is nonlinear (alpha = 0.5): E^{1/2} point-wise (what the shortcut produces) to 1e-11, f at the probes to 1e-10.
    The bound on f is north_star's one-step tolerance, not 1e-11: at 128^3, r = 15 this configuration amplifies rounding by
    ~1e5 through the ill-conditioned first QRs - two builds of the SAME algorithm that differ only in summation order (the
    CTA-tile and the warp-autonomous sub-flow-1 kernel) differ by 3-6e-11 in f after these 3 steps and by 1.9e-10 in
    E^{1/2} after one, while shortcut and flow agree to 1.5e-15 in E^{1/2} after one step and 8e-13 after three (measured
    on B200, reading R18)."""
    from paper_2110_13481_b200 import dlr
    for n, r, nsteps in ((64, 10, 6), (128, 15, 3)):
        cfg = inputs.make_config(4, n_x=n, n_v=n, r=r)
        X, S, V = inputs.initial_factors(cfg)
        ix, iv = inputs.probe_indices(cfg)
        res = []
        for flags in (0, dlr.FLAG_PREDICTOR_L_FLOW):
            ctx = make_ctx(cfg, flags=flags)
            ctx.set_initial(X, S, V)
            ctx.run(cfg["tau"], nsteps)
            m, f = ctx.moments(ix, iv)
            res.append((ctx.get_field(), f, m))
            ctx.close()
        (Ea, fa, ma), (Eb, fb, mb) = res
        assert np.abs(Ea - Eb).max() <= 1e-11 * np.abs(Eb).max(), (n, r)
        assert np.abs(fa - fb).max() <= 1e-10 * np.abs(fb).max(), (n, r)
        assert rel(ma["electric_energy"], mb["electric_energy"]) <= 1e-11


def test_config4_one_step():
    """BASELINE.json config 4 (128^3 x 128^3, r = 15, alpha = 0.5: stresses the real-space terms and the QR) at full
    size: one step against the oracle run live (about a minute of host time)."""
    cfg = inputs.make_config(4)
    gx, gv = grids(cfg)
    X, S, V = inputs.initial_factors(cfg)
    ix, iv = inputs.probe_indices(cfg)
    ctx = make_ctx(cfg)
    ctx.set_initial(X, S, V)
    ctx.step(cfg["tau"])
    X, S, V = O.step_alg2(X, S, V, cfg["tau"], gx, gv)
    check(ctx, X, S, V, gx, gv, ix, iv, TOL_STEP)
    ctx.close()


def test_config5_invariants():
    """BASELINE.json config 5 (256^3 x 256^3, r = 20, band-limited rank-20 perturbation) at full size, in the launch
    configuration bench.py times: properties that hold at any size (an oracle step here needs ~30 GB and minutes):
    the bases stay orthonormal, the mass follows the closed form L^3 up to the low-rank drift bound of SURVEY P10,
    ||S||_F moves by O(tau^2)-small amounts, no QR repair, nothing non-finite."""
    import torch
    cfg = inputs.make_config(5)
    X, S, V = inputs.initial_factors(cfg)
    ctx = make_ctx(cfg)
    ctx.set_initial(X, S, V)
    del X, V
    m0 = ctx.moments()
    for _ in range(3):
        ctx.step(cfg["tau"])
    m = ctx.moments()
    assert m["qr_fallbacks"] == 0 and m["nonfinite"] == 0
    assert rel(m0["mass"], (4 * math.pi) ** 3) <= 1e-7
    assert rel(m["mass"], m0["mass"]) <= 1e-6
    assert rel(m["s_fro"], m0["s_fro"]) <= 1e-4
    assert rel(m["kinetic_energy"], m0["kinetic_energy"]) <= 1e-4
    Xg, Sg, Vg = ctx.get_factors()
    r = cfg["r"]
    hx3 = ((cfg["x_hi"] - cfg["x_lo"]) / cfg["n_x"]) ** 3
    hv3 = ((cfg["v_hi"] - cfg["v_lo"]) / cfg["n_v"]) ** 3
    for A, h3 in ((Xg, hx3), (Vg, hv3)):
        At = torch.from_numpy(A)
        G = (At.T @ At).numpy() * h3
        assert np.abs(G - np.eye(r)).max() < 1e-11
    ctx.close()


def test_bit_reproducible_and_reinitialisable():
    """all reductions are fixed-order (per-CTA rows, group sums, single-CTA consumers; no atomics on data), so two
    contexts fed the same inputs agree BIT FOR BIT; the same holds for one context after dlr_set_initial is called
    again (the cached C coefficients, the warm-started eigenvectors and the step graph must not leak state)."""
    cfg = inputs.make_config(1, n=16, r=10)
    X, S, V = inputs.initial_factors(cfg)
    a, b = make_ctx(cfg), make_ctx(cfg)
    outs = []
    for ctx in (a, b):
        ctx.set_initial(X, S, V)
        for _ in range(4):
            ctx.step(cfg["tau"])
        outs.append(ctx.get_factors())
    for u, w in zip(*outs):
        assert np.array_equal(u, w)
    a.set_initial(X, S, V)                       # again on a used context
    for _ in range(4):
        a.step(cfg["tau"])
    for u, w in zip(a.get_factors(), outs[0]):
        assert np.array_equal(u, w)
    a.close()
    b.close()


def test_step_size_change_recaptures_the_graph():
    """tau may change from call to call (the step graph is re-captured and the tables rebuilt): steps of size
    tau, tau/2, tau/2, tau against the oracle doing the same"""
    cfg = inputs.make_config(1, n=16, r=8)
    gx, gv = grids(cfg)
    X, S, V = inputs.initial_factors(cfg)
    ix, iv = inputs.probe_indices(cfg)
    ctx = make_ctx(cfg)
    ctx.set_initial(X, S, V)
    for tau in (0.1, 0.05, 0.05, 0.1):
        ctx.step(tau)
        X, S, V = O.step_alg2(X, S, V, tau, gx, gv)
        check(ctx, X, S, V, gx, gv, ix, iv, TOL_STEP)
    ctx.close()


def test_strongly_anisotropic_grids():
    """n_x << n_v and n_x >> n_v (the paper's headline shape is 64^3 x 256^3): different tile shapes,
    tables and FFT plans on the two grids inside one step; both orders"""
    for n_x, n_v, order in ((8, 32, 2), (32, 8, 2), (8, 32, 1)):
        cfg = inputs.make_config(2, n_x=n_x, n_v=n_v, r=8)
        gx, gv = grids(cfg)
        X, S, V = inputs.initial_factors(cfg)
        ix, iv = inputs.probe_indices(cfg)
        ctx = make_ctx(cfg, order)
        ctx.set_initial(X, S, V)
        step = O.step_alg2 if order == 2 else O.step_alg1
        for _ in range(2):
            ctx.step(0.1)
            X, S, V = step(X, S, V, 0.1, gx, gv)
            check(ctx, X, S, V, gx, gv, ix, iv, TOL_STEP)
        ctx.close()


def _run_to(cfg, order, nsteps, T, ix, iv, X, S, V):
    ctx = make_ctx(cfg, order)
    ctx.set_initial(X, S, V)
    ctx.run(T / nsteps, nsteps)
    m, f = ctx.moments(ix, iv)
    ctx.close()
    assert m["qr_fallbacks"] == 0 and m["nonfinite"] == 0
    return f


def test_paper_convergence_orders_at_full_size():
    """Section 6.1 of the paper at its own size (Fig. 3 left): linear Landau, 32^3 x 32^3, r = 10, T = 1;
    error in maximum norm at the final time (here over 4096 seeded probe pairs) against a fine reference (Algorithm 2,
    2000 steps) for 40 and 80 steps: Algorithm 1 converges at order 1, Algorithm 2 at order 2.  Runs on the GPU path
    only (the oracle pins the same orders at n = 8, tests/test_oracle_physics.py)."""
    cfg = inputs.make_config(2)
    X, S, V = inputs.initial_factors(cfg)
    ix, iv = inputs.probe_indices(cfg, nprobe=4096, seed=11)
    ref = _run_to(cfg, 2, 2000, 1.0, ix, iv, X, S, V)
    err = {}
    for order in (1, 2):
        for m in (40, 80):
            f = _run_to(cfg, order, m, 1.0, ix, iv, X, S, V)
            err[order, m] = np.abs(f - ref).max() / np.abs(ref).max()
    assert 1.7 < err[1, 40] / err[1, 80] < 2.4, err
    assert 3.3 < err[2, 40] / err[2, 80] < 5.0, err
    assert err[2, 80] < 0.1 * err[1, 80], err


def test_paper_linear_landau_headline_shape():
    """Section 6.2 of the paper (Fig. 4): linear Landau damping on 64^3 x 256^3, r = 10, tau = 0.1 up
    to T = 60 (600 steps of Algorithm 2).  The electric energy decays at the theoretical rate (-0.1533 for k = 0.5,
    BASELINE.json; fitted on the maxima up to t = 25), falls by more than four orders of magnitude, mass and total
    energy are conserved to the levels the paper reports (3e-8 and 7e-7; bounds here 1e-6 and 1e-5)."""
    cfg = inputs.make_config(2, n_x=64, n_v=256)
    X, S, V = inputs.initial_factors(cfg)
    ctx = make_ctx(cfg)
    ctx.set_initial(X, S, V)
    del X, V
    tau, nsteps = 0.1, 600
    m0 = ctx.moments()
    ee, mass_err, en_err = [m0["electric_energy"]], 0.0, 0.0
    e0 = m0["kinetic_energy"] + m0["electric_energy"]
    for _ in range(nsteps):
        ctx.step(tau)
        m = ctx.moments()
        ee.append(m["electric_energy"])
        mass_err = max(mass_err, rel(m["mass"], m0["mass"]))
        en_err = max(en_err, rel(m["kinetic_energy"] + m["electric_energy"], e0))
    assert m["qr_fallbacks"] == 0 and m["nonfinite"] == 0
    ctx.close()
    ee = np.array(ee)
    tp, lp = [], []
    for i in range(1, len(ee) - 1):
        if ee[i] > ee[i - 1] and ee[i] > ee[i + 1] and tau * i < 25.0:
            tp.append(tau * i)
            lp.append(math.log(ee[i]))
    gamma = 0.5 * np.polyfit(tp, lp, 1)[0]
    print(f"gamma = {gamma:.4f}, min ee / ee0 = {ee.min() / ee[0]:.2e}, mass err = {mass_err:.2e}, energy err = {en_err:.2e}")
    assert gamma == pytest.approx(-0.1533, rel=0.04)
    assert ee.min() < 1e-4 * ee[0]
    assert mass_err < 1e-6
    assert en_err < 1e-5


def test_paper_two_stream_initial_value():
    """the paper's own two-stream initial value, eq. (21) (inputs config 6): beams at different
    velocities in all three directions, so every momentum component and all three real-space terms are exercised.
    Closed forms at t = 0 (mass L^3, momentum = mean beam velocity x mass), then two steps against the oracle."""
    cfg = inputs.make_config(6, n=16, r=10, tau=0.01)
    gx, gv = grids(cfg)
    X, S, V = inputs.initial_factors(cfg)
    ix, iv = inputs.probe_indices(cfg)
    ctx = make_ctx(cfg)
    ctx.set_initial(X, S, V)
    m = ctx.moments()
    mass = (10 * math.pi) ** 3
    assert rel(m["mass"], mass) <= 1e-5                      # 16-point quadrature of the Gaussians
    for d, vmean in enumerate((0.0, -1.125, -1.0)):
        assert abs(m["momentum"][d] - vmean * mass) <= 1e-4 * mass
    for _ in range(2):
        ctx.step(cfg["tau"])
        X, S, V = O.step_alg2(X, S, V, cfg["tau"], gx, gv)
        check(ctx, X, S, V, gx, gv, ix, iv, TOL_STEP)
    ctx.close()


def test_paper_two_stream_instability_128():
    """Section 6.3 of the paper (Fig. 5): two-stream instability (eq. (21)) on 128^3 x 128^3, r = 10,
    tau = 0.06 up to T = 60 (1000 steps of Algorithm 2).  The paper prints no numbers, only the behaviour: "the electric
    energy shows an exponential increase before entering into a saturation phase", mass and energy errors grow in the
    nonlinear phase.  Checked here: growth by more than four orders of magnitude that is exponential (straight in
    log scale over t in [15, 30]), saturation afterwards, no QR repair, nothing non-finite; mass and total energy
    conserved to 1e-3 up to the onset of saturation (t <= 30; measured 2e-5).  After that the rank-10 dynamics is chaotic: two builds
    of this library that differ only in rounding order agree to 4-5 digits up to t = 42 and then drift apart, so the
    late phase is only required to stay bounded (electric energy within a factor 5, conservation errors < 0.1)."""
    cfg = inputs.make_config(6, n_x=128, n_v=128, r=10)
    X, S, V = inputs.initial_factors(cfg)
    ctx = make_ctx(cfg)
    ctx.set_initial(X, S, V)
    del X, V
    tau, nsteps = 0.06, 1000
    m0 = ctx.moments()
    e0 = m0["kinetic_energy"] + m0["electric_energy"]
    t, ee, worst, worst_early = [], [], 0.0, 0.0
    for i in range(1, nsteps + 1):
        ctx.step(tau)
        if i % 10 == 0:
            m = ctx.moments()
            t.append(i * tau)
            ee.append(m["electric_energy"])
            werr = max(rel(m["mass"], m0["mass"]), rel(m["kinetic_energy"] + m["electric_energy"], e0))
            worst = max(worst, werr)
            if i * tau <= 30.0:
                worst_early = max(worst_early, werr)
            assert m["qr_fallbacks"] == 0 and m["nonfinite"] == 0
    ctx.close()
    t, ee = np.array(t), np.array(ee)
    assert ee.max() > 1e4 * ee[t < 10].min()
    lin = (t >= 15) & (t <= 30)
    slope, icpt = np.polyfit(t[lin], np.log(ee[lin]), 1)
    assert 0.3 < slope < 0.7
    assert np.abs(np.log(ee[lin]) - (slope * t[lin] + icpt)).max() < 0.5          # exponential growth
    sat = ee[t > 36]
    assert sat.max() < 5.0 * sat.min()                                             # saturation
    assert worst_early < 1e-3
    assert worst < 0.1


def test_error_codes():
    from paper_2110_13481_b200 import dlr
    cfg = inputs.make_config(1)
    with pytest.raises(dlr.DlrError) as e:
        dlr.dlr_workspace_bytes(dlr.make_config(12, 8, 0, 1, -1, 1, 5))
    assert e.value.code == -2
    with pytest.raises(dlr.DlrError) as e:
        dlr.dlr_workspace_bytes(dlr.make_config(8, 8, 0, 1, -1, 1, 7))
    assert e.value.code == -2
    ctx = make_ctx(cfg)
    with pytest.raises(dlr.DlrError) as e:
        ctx.step(0.1)
    assert e.value.code == -6
    X, S, V = inputs.initial_factors(cfg)
    with pytest.raises(dlr.DlrError) as e:
        ctx.set_initial(1.001 * X, S, V)
    assert e.value.code == -5
    ctx.set_initial(X, S, V)
    ctx.step(0.1)
    assert ctx.launches_per_step() > 0
    ctx.close()

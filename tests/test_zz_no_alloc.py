"""dlr_probe_noalloc (include/dlr.h): f = X S V^T at probes through a static device scratch array, no device
allocation, against the existing path (the probes of dlr_moments, which use the context's workspace).  Collected last
on purpose (file name): the suite runs with pytest -x."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _device_factors(torch, dlr, ctx):
    """the context's current factors as device tensors in the ABI layout (row c = column c of the factor)"""
    X = torch.empty((ctx.r, ctx.Nx), dtype=torch.float64, device=ctx.device)
    S = torch.empty((ctx.r, ctx.r), dtype=torch.float64, device=ctx.device)
    V = torch.empty((ctx.r, ctx.Nv), dtype=torch.float64, device=ctx.device)
    rc = dlr.lib().dlr_get_factors(ctx.h, X.data_ptr(), S.data_ptr(), V.data_ptr(), 1)
    assert rc == 0
    return X, S, V


def test_probe_noalloc_matches_moments_probes_twice_in_a_row():
    import torch
    from paper_2110_13481_b200 import dlr, inputs
    cfg = inputs.make_config(1, n=16, r=10)
    ctx = dlr.Dlr(dlr.config_from_inputs(cfg), device="cuda:0")
    ctx.set_initial(*inputs.initial_factors(cfg))
    ctx.step(cfg["tau"])
    ctx.step(cfg["tau"])
    X, S, V = _device_factors(torch, dlr, ctx)
    torch.cuda.synchronize()
    free0 = None
    # two calls in a row with different probe sets and sizes: the second must not see anything of the first
    for call, (nprobe, seed) in enumerate(((1000, 7), (64, 11), (dlr.NOALLOC_MAX_PROBES, 13))):
        ix, iv = inputs.probe_indices(cfg, nprobe=nprobe, seed=seed)
        _, f_ref = ctx.moments(ix, iv)                         # existing path: workspace scratch
        f = dlr.probe_noalloc(X, S, V, ix, iv)
        assert np.isfinite(f).all()
        err = np.abs(f - f_ref).max() / np.abs(f_ref).max()
        assert err <= 1e-12, (call, err)                       # the tests' tolerance is 1e-10; same arithmetic here
        if call == 0:                                          # after the first call (module load, symbol look-up) ...
            free0 = torch.cuda.mem_get_info(0)[0]
    assert torch.cuda.mem_get_info(0)[0] >= free0              # ... no call takes device memory
    ctx.close()


def test_probe_noalloc_rejects_what_the_scratch_cannot_hold():
    import torch
    from paper_2110_13481_b200 import dlr
    L = dlr.lib()
    r, N = 5, 512
    X = torch.zeros((r, N), dtype=torch.float64, device="cuda:0")
    S = torch.zeros((r, r), dtype=torch.float64, device="cuda:0")
    n = dlr.NOALLOC_MAX_PROBES + 1
    with pytest.raises(dlr.DlrError) as e:
        dlr.probe_noalloc(X, S, X, np.zeros(n, dtype=np.int64), np.zeros(n, dtype=np.int64))
    assert e.value.code == -7 and "DLR_NOALLOC_MAX_PROBES" in str(e.value)
    assert L.dlr_strerror(-7).decode().startswith("size exceeds")
    with pytest.raises(dlr.DlrError) as e:                     # an index outside the grid never reaches the kernel
        dlr.probe_noalloc(X, S, X, np.array([N]), np.array([0]))
    assert e.value.code == -1
    f = dlr.probe_noalloc(X, S, X, np.array([3, 4]), np.array([0, N - 1]))   # still usable after the errors
    assert (f == 0.0).all()
    assert L.dlr_noalloc_last_error() == b""

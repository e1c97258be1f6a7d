"""cf_mppi_update_static -- the planner update for callers that cannot allocate device memory -- against cf_mppi_update.

Who this entry point is for (include/cf.h has the full text): a planning thread inside a fixed-rate control loop, which
must not call cudaMalloc once it runs (the call takes driver locks and can stall the device past the deadline), and code
that lives under someone else's memory pool (a plug-in, a framework with a fixed arena) and gets input / output buffers
but nothing else.  For them the scratch of the update kernel is an 8 MiB array built into libcf.so, one per GPU, shared by
every simulator and never cleared between calls.

What is checked: two calls in a row on the same simulator state give what the caller-scratch path gives -- elite index
sets, thresholds, minimum costs and the best controller bit for bit (integer / bit-pattern work), scores, weight sums,
plan and warm-started nominal within the tolerances tests/test_gpu_mppi.py uses for the same quantities (2e-5 relative,
5e-6 absolute) -- although the second call finds the first one's leftovers in the array (the first is made with more
elites and a longer horizon than the second, so the leftovers cover and exceed what the second one writes); and that a
request beyond the array's size is refused before anything is launched.

The file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It passes alone in a fresh process (the first call does the per-device address look-up) and after the
other GPU tests.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _sim_after_rollout(cf, wl, nominal_np):
    """A simulator in the state cf_mppi_update expects: reset, broadcast start state, ONE rollout of horizon * cmd_hold steps."""
    import torch
    g = cf.Sim(wl.M, 1, wl.model, wl.params)
    g.reset(wl.seed)
    g.set_state(wl.broadcast_state.astype(np.float32), broadcast=True)
    g.step(torch.as_tensor(nominal_np, device="cuda"), wl.n_steps, cmd_hold=wl.cmd_hold)
    return g


def _nominal(wl, seed):
    rng = np.random.default_rng(seed)
    nom = wl.cmds.copy()
    nom[..., :2] += rng.uniform(-0.2, 0.2, nom[..., :2].shape).astype(np.float32)
    nom[..., 3] += rng.uniform(-0.03, 0.03, nom[..., 3].shape).astype(np.float32)
    return nom


def _compare(static, ref, n_ctrl):
    """static / ref: dicts of numpy arrays (elites, info, plan, nominal) from the two paths."""
    assert np.array_equal(static["elites"], ref["elites"])                                  # index work: exact
    si, ri = static["info"], ref["info"]
    assert np.array_equal(si[1:4 * n_ctrl:4], ri[1:4 * n_ctrl:4])                           # J_min: a selected input value
    assert np.array_equal(si[3:4 * n_ctrl:4], ri[3:4 * n_ctrl:4])                           # threshold cost: likewise
    assert si.view(np.int32)[4 * n_ctrl] == ri.view(np.int32)[4 * n_ctrl]                   # best controller
    np.testing.assert_allclose(si[0:4 * n_ctrl:4], ri[0:4 * n_ctrl:4], rtol=2e-5)           # score S_c
    np.testing.assert_allclose(si[2:4 * n_ctrl:4], ri[2:4 * n_ctrl:4], rtol=2e-5)           # sum of weights
    np.testing.assert_allclose(static["plan"], ref["plan"], rtol=0, atol=5e-6)
    np.testing.assert_allclose(static["nominal"], ref["nominal"], rtol=0, atol=5e-6)


def _run_both(cf, W, *, seed, n_ctrl, worlds_per_ctrl, horizon, cmd_hold, n_elite, lam, shift):
    import torch
    wl = W.mppi(seed=seed, n_ctrl=n_ctrl, worlds_per_ctrl=worlds_per_ctrl, horizon=horizon, cmd_hold=cmd_hold,
                n_elite=n_elite)
    nom_np = _nominal(wl, seed)
    g = _sim_after_rollout(cf, wl, nom_np)
    mp = g.mppi_params(horizon, cmd_hold, n_elite, lam, shift)

    # existing path: scratch allocated by the binding (a torch tensor), passed to cf_mppi_update
    nom_ref = torch.as_tensor(nom_np, device="cuda")
    out = g.mppi_update(mp, nom_ref, want_elites=True)
    ref = {k: out[k].cpu().numpy().copy() for k in ("elites", "info", "plan")}
    ref["nominal"] = nom_ref.cpu().numpy()

    # new path: the caller brings inputs and outputs only; the update does not advance the simulator, so it can be repeated
    nom_st = torch.as_tensor(nom_np, device="cuda")
    plan = torch.full((horizon, 4), float("nan"), dtype=torch.float32, device="cuda")
    info = torch.full((4 * n_ctrl + 4,), float("nan"), dtype=torch.float32, device="cuda")
    elites = torch.full((n_ctrl, n_elite), -1, dtype=torch.int32, device="cuda")
    g.mppi_update_static(mp, nom_st, plan, info, elites)
    torch.cuda.synchronize()
    static = dict(elites=elites.cpu().numpy(), info=info.cpu().numpy(), plan=plan.cpu().numpy(), nominal=nom_st.cpu().numpy())
    _compare(static, ref, n_ctrl)
    return static


def test_static_scratch_update_matches_the_caller_scratch_update_on_two_calls_in_a_row():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2606_01478_b200 import build, cf, workloads as W
    build.build()
    # call 1: 3 controllers x 64 elites x 9 knots -- fills 3 x 64 x 10 rows of the shared array
    a = _run_both(cf, W, seed=31, n_ctrl=3, worlds_per_ctrl=211, horizon=9, cmd_hold=4, n_elite=64, lam=0.5, shift=1)
    # call 2, straight after it: a different, SMALLER problem (2 x 11 x 6) -- every byte it uses still holds call 1's data
    b = _run_both(cf, W, seed=32, n_ctrl=2, worlds_per_ctrl=384, horizon=5, cmd_hold=3, n_elite=11, lam=0.05, shift=2)
    assert a["plan"].shape == (9, 4) and b["plan"].shape == (5, 4)
    assert np.isfinite(a["plan"]).all() and np.isfinite(b["plan"]).all()                   # the NaN fill was overwritten


def test_static_scratch_update_repeated_on_one_simulator_gives_the_same_bits():
    """The same update twice on the same simulator state and stream: identical output, i.e. nothing of the first call
    (completion counter included) leaks into the second."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2606_01478_b200 import build, cf, workloads as W
    build.build()
    wl = W.mppi(seed=33, n_ctrl=3, worlds_per_ctrl=500, horizon=6, cmd_hold=5, n_elite=25)
    nom_np = _nominal(wl, 5)
    g = _sim_after_rollout(cf, wl, nom_np)
    mp = g.mppi_params(6, 5, 25, 0.5, 1)
    outs = []
    for _ in range(2):
        nom = torch.as_tensor(nom_np, device="cuda")
        plan = torch.empty((6, 4), dtype=torch.float32, device="cuda")
        info = torch.empty(16, dtype=torch.float32, device="cuda")
        elites = torch.empty((3, 25), dtype=torch.int32, device="cuda")
        g.mppi_update_static(mp, nom, plan, info, elites)
        torch.cuda.synchronize()
        # info: 4 n_ctrl + 1 words are defined (the 3 words of padding after the best-controller index are never written)
        outs.append([t.cpu().numpy().copy() for t in (nom, plan, info[:13], elites)])
    for x, y in zip(*outs):
        assert np.array_equal(x.view(np.uint32) if x.dtype == np.float32 else x, y.view(np.uint32) if y.dtype == np.float32 else y)


def test_static_scratch_update_refuses_what_does_not_fit():
    """4 controllers x 4096 elites x 60 knots need 16 MB of scratch: CF_E_BUFFER, outputs untouched."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2606_01478_b200 import build, cf, workloads as W
    build.build()
    wl = W.mppi(seed=34, n_ctrl=4, worlds_per_ctrl=4200, horizon=60, cmd_hold=1, n_elite=4096)
    nom_np = _nominal(wl, 6)
    g = _sim_after_rollout(cf, wl, nom_np)
    mp = g.mppi_params(60, 1, 4096, 0.5, 1)
    nom = torch.as_tensor(nom_np, device="cuda")
    plan = torch.full((60, 4), 7.0, dtype=torch.float32, device="cuda")
    info = torch.full((20,), 7.0, dtype=torch.float32, device="cuda")
    with pytest.raises(cf.CfError) as e:
        g.mppi_update_static(mp, nom, plan, info)
    assert e.value.code == -4 and "8388608" in str(e.value)                                # CF_E_BUFFER, the limit is named
    torch.cuda.synchronize()
    assert (plan.cpu().numpy() == 7.0).all() and (info.cpu().numpy() == 7.0).all()
    assert np.array_equal(nom.cpu().numpy(), nom_np)
    out = g.mppi_update(mp, nom, want_elites=False)                                        # the caller-scratch path still takes it
    assert np.isfinite(out["plan"].cpu().numpy()).all()

"""Adaptive RKF45 stepping (mm_rkf45_*) against the oracle's O10, through the C ABI:
every attempt's error estimate, accept/reject decision and next step size, and the trajectory."""
import numpy as np
import pytest
import torch

import workloads as w
from gpu_util import make_ctx, make_problem, round_input, to_dev

pytestmark = pytest.mark.gpu

TRAJ_TOL = {"f64": 1e-10, "f32": 1e-4}      # BASELINE.json north_star, in m
ERR_RTOL = {"f64": 1e-7, "f32": 2e-3}       # relative agreement of the error estimates


def drive(oracle, cfg, dt, attempts, tol, dt0, dt_min=0.0, dt_max=1.0):
    m, m64 = round_input(cfg.initial_m(), dt)
    P = make_problem(oracle, cfg)
    ctx = make_ctx(cfg, dt)
    md = to_dev(m)
    ctx.rkf45_init(t0=0.0, dt0=dt0, tol=tol, dt_min=dt_min, dt_max=dt_max)
    ref, t_ref, dt_ref = m64, 0.0, dt0
    n_acc = n_rej = 0
    for a in range(attempts):
        ctx.rkf45_step(md)
        ref, err, acc, dt_next = P.rkf45_step(ref, dt_ref, tol, dt_min, dt_max)
        if acc:
            t_ref += dt_ref
            n_acc += 1
        else:
            n_rej += 1
        st = ctx.rkf45_state()
        assert st["accepted"] == acc, (a, st, err)
        assert abs(st["err"] - err) <= ERR_RTOL[dt] * err, (a, st["err"], err)
        assert abs(st["dt_last"] - dt_ref) <= 1e-3 * dt_ref
        assert abs(st["dt_next"] - dt_next) <= ERR_RTOL[dt] * dt_next, (a, st["dt_next"], dt_next)
        assert abs(st["t"] - t_ref) <= 1e-3 * max(t_ref, dt0)
        assert w.traj_error(md.cpu().numpy(), ref) <= TRAJ_TOL[dt], a
        dt_ref = dt_next
    assert (st["n_accepted"], st["n_rejected"]) == (n_acc, n_rej)
    assert abs(np.linalg.norm(md.cpu().numpy(), axis=-1) - 1).max() < (1e-14 if dt == "f64" else 1e-6)
    ctx.close()
    return n_acc, n_rej


@pytest.mark.parametrize("dt", ["f64", "f32"])
def test_rkf45_config1_attempts(oracle, dt):
    """Config 1 (16x16x2, demag + exchange, alpha = 0.5, random m): the first attempt at 4e-13 s is
    rejected against tol = 1e-6 and the controller settles; every attempt is compared."""
    tol = 1e-6 if dt == "f64" else 1e-5
    n_acc, n_rej = drive(oracle, w.get_config(1), dt, attempts=14, tol=tol, dt0=4e-13)
    assert n_acc >= 8 and n_rej >= 1


@pytest.mark.parametrize("dt", ["f64", "f32"])
def test_rkf45_config2_strip(oracle, dt):
    """Config 2 (SP4-shaped strip with the Zeeman field): 40 attempts from dt0 = 1e-13 s."""
    tol = 1e-7 if dt == "f64" else 1e-5
    n_acc, _ = drive(oracle, w.get_config(2), dt, attempts=40, tol=tol, dt0=1e-13, dt_max=5e-13)
    assert n_acc >= 30


def test_rkf45_clamps_and_rejection_leaves_m(oracle):
    cfg = w.get_config(1)
    ctx = make_ctx(cfg, "f64")
    m = to_dev(cfg.initial_m())
    m_before = m.clone()
    ctx.rkf45_init(dt0=2e-13, tol=1e-30, dt_min=1e-13, dt_max=1e-12)     # impossible tolerance
    ctx.rkf45_step(m)
    st = ctx.rkf45_state()
    assert not st["accepted"] and st["n_rejected"] == 1 and st["t"] == 0.0
    assert st["dt_next"] == 1e-13                                       # 0.2 x dt clamped to dt_min
    assert torch.equal(m, m_before)
    ctx.rkf45_init(dt0=2e-13, tol=1.0, dt_min=1e-13, dt_max=3e-13)
    ctx.rkf45_step(m)
    st = ctx.rkf45_state()
    assert st["accepted"] and st["dt_next"] == 3e-13 and st["t"] == 2e-13
    assert not torch.equal(m, m_before)
    ctx.close()


def test_rkf45_needs_init_and_validates():
    from paper_2606_01114_b200 import Context, MMError
    ctx = Context((8, 8, 2), (1e-9,) * 3, dtype=torch.float32)
    ctx.set_material(8e5, 1.3e-11, 0.0, (0, 0, 1), 0.1)
    ctx.set_terms(2)
    m = torch.zeros(8, 8, 2, 3, device="cuda")
    with pytest.raises(MMError) as e:
        ctx.rkf45_step(m)
    assert e.value.status == 3
    for bad in (dict(dt0=0.0), dict(tol=0.0), dict(dt0=1e-13, dt_min=2e-13), dict(dt0=1e-13, dt_max=1e-14)):
        with pytest.raises(MMError) as e:
            ctx.rkf45_init(**bad)
        assert e.value.status == 1
    ctx.close()


def test_rkf45_attempt_is_graph_capturable(oracle):
    """No host round trip inside an attempt: a captured CUDA graph of one attempt, replayed,
    follows the same trajectory as eager attempts."""
    cfg = w.get_config(1)
    m0 = cfg.initial_m()
    outs = []
    for use_graph in (False, True):
        ctx = make_ctx(cfg, "f64")
        m = to_dev(m0)
        ctx.rkf45_init(dt0=1e-13, tol=1e-7)
        if use_graph:
            s = torch.cuda.Stream()
            s.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(s):
                ctx.use_current_stream()
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=s):
                    ctx.rkf45_step(m)
                for _ in range(5):          # the capture itself enqueued nothing
                    g.replay()
            s.synchronize()
        else:
            for _ in range(5):
                ctx.rkf45_step(m)
        st = ctx.rkf45_state()
        outs.append((m.cpu().numpy().copy(), st["t"], st["n_accepted"]))
        ctx.close()
    assert outs[0][1] == outs[1][1] and outs[0][2] == outs[1][2]
    assert np.array_equal(outs[0][0], outs[1][0])


def test_controller_state_survives_a_later_demag_init(oracle):
    """mm_rkf45_init and mm_minimize_init BEFORE the first mm_demag_init (the header fixes no order): the
    table upload of mm_demag_init must not clear the device-resident controller records."""
    from paper_2606_01114_b200 import Context
    cfg = w.get_config(1)
    ctx = Context(cfg.n, cfg.d, dtype=torch.float64)
    ctx.set_material(cfg.Ms, cfg.Aex, cfg.Ku, cfg.axis, cfg.alpha, cfg.gamma)
    ctx.set_terms(cfg.terms)
    ctx.rkf45_init(t0=0.0, dt0=2e-13, tol=1e-6, dt_min=0.0, dt_max=1e-12)
    ctx.minimize_init(tau0=1e-7, tau_min=1e-10, tau_max=1e-4, tol=1e-9)
    ctx.demag_init()
    st = ctx.rkf45_state()
    assert st["dt_next"] == 2e-13 and st["t"] == 0.0
    m, m64 = round_input(cfg.initial_m(), "f64")
    md = to_dev(m)
    ctx.rkf45_step(md)
    ref, err, acc, dt_next = make_problem(oracle, cfg).rkf45_step(m64, 2e-13, 1e-6, 0.0, 1e-12)
    st = ctx.rkf45_state()
    assert st["dt_last"] == 2e-13 and st["accepted"] == acc and abs(st["err"] - err) <= 1e-7 * err
    assert w.traj_error(md.cpu().numpy(), ref) <= TRAJ_TOL["f64"]
    md2 = to_dev(m)
    ctx.minimize_step(md2)
    n_it, tau, dm, conv = ctx.minimize_state()
    assert n_it == 1 and tau == 1e-7 and dm > 0
    ctx.close()


def test_rkf45_non_finite_state_is_rejected_not_accepted():
    """A blown-up state (NaN in m) must not read as err = 0 and be accepted with dt * 5."""
    cfg = w.get_config(1)
    ctx = make_ctx(cfg, "f64")
    m = cfg.initial_m()
    m[3, 4, 1, :] = np.nan
    md = to_dev(m)
    ctx.rkf45_init(t0=0.0, dt0=1e-13, tol=1e-6)
    ctx.rkf45_step(md)
    st = ctx.rkf45_state()
    assert not st["accepted"] and st["err"] == np.inf and st["dt_next"] == pytest.approx(0.2e-13)
    ctx.close()

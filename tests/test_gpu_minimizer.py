"""Barzilai-Borwein minimiser (reading Q30): the device-resident iteration
against the oracle's O13, iteration by iteration (state m, step length, maximum change, stop flag),
and the equilibria the minimiser must reach."""
import numpy as np
import pytest
import torch

import workloads as w
from gpu_util import TRAJ_TOL, make_ctx, make_problem, round_input, to_dev

pytestmark = pytest.mark.gpu
MU0 = 4e-7 * np.pi


def cfg_for(n, d, **kw):
    base = w.get_config(1)
    return w.Config(**{**base.__dict__, "n": n, "d": d, "name": "t", **kw})


@pytest.mark.parametrize("dt", ["f64", "f32"])
@pytest.mark.parametrize("n,d,terms", [((16, 16, 2), (5e-9, 5e-9, 3e-9), 1 | 2), ((100, 25, 1), (5e-9, 5e-9, 3e-9), 1 | 2),
                                       ((12, 10, 6), (2e-9, 2e-9, 2e-9), 1 | 2 | 8), ((32, 16, 8), (4e-9, 3e-9, 2e-9), 2 | 8)])
def test_iterations_match_oracle(oracle, n, d, terms, dt):
    """PAPER.md:146-148 minimises [demag, exchange] on the SP4 strip; 30 iterations from a smooth state."""
    cfg = cfg_for(n, d, terms=terms, Hext=(2e4, 1e4, 3e4))
    m0 = w.box_filter_renormalise(w.random_unit_vectors(707, n))
    m, m64 = round_input(m0, dt)
    P = make_problem(oracle, cfg)
    tau0, tmin, tmax, tol = 2e-7, 1e-10, 1e-4, 1e-9
    bb = oracle.BBMinimizer(P, m64, tau0=tau0, tau_min=tmin, tau_max=tmax, tol=tol)
    ctx = make_ctx(cfg, dt)
    ctx.minimize_init(tau0, tmin, tmax, tol)
    md = to_dev(m)
    rtol = 1e-7 if dt == "f64" else 5e-3
    for it in range(30):
        tau_o, dm_o, conv_o = bb.step()
        ctx.minimize_step(md)
        nit, tau_g, dm_g, conv_g = ctx.minimize_state()
        assert nit == it + 1 and conv_g == conv_o
        assert abs(tau_g - tau_o) <= rtol * tau_o, (it, tau_g, tau_o)
        assert abs(dm_g - dm_o) <= rtol * dm_o + 1e-12, (it, dm_g, dm_o)
        assert w.traj_error(md.cpu().numpy(), bb.m) <= TRAJ_TOL[dt], it
    nrm = md.double().norm(dim=-1)
    assert float((nrm - 1).abs().max()) < (1e-13 if dt == "f64" else 1e-5)


@pytest.mark.parametrize("dt", ["f64", "f32"])
def test_stoner_wohlfarth_and_coordinated_stop(oracle, dt):
    """Uniform block, anisotropy along z, hard-axis field h H_k: every cell ends at m_x = h; after the
    stop flag is raised further iterations leave m and the counter untouched."""
    n, d, Ms, Ku, h = (8, 4, 4), (2e-9,) * 3, 8e5, 5e5, 0.5
    Hk = 2 * Ku / (MU0 * Ms)
    cfg = cfg_for(n, d, Ms=Ms, Ku=Ku, axis=(0.0, 0.0, 1.0), Hext=(h * Hk, 0.0, 0.0), terms=2 | 4 | 8)
    m0 = np.zeros(n + (3,))
    m0[...] = np.array([np.sin(0.3) * np.cos(0.7), np.sin(0.3) * np.sin(0.7), np.cos(0.3)])
    m, _ = round_input(m0, dt)
    ctx = make_ctx(cfg, dt)
    tol = 1e-13 if dt == "f64" else 1e-7
    ctx.minimize_init(1e-7, 1e-9, 1e-3, tol)
    md = to_dev(m)
    nit, conv = ctx.minimize(md, max_iter=500, check_every=7)
    assert conv and nit < 300
    got = md.double().cpu().numpy()
    assert np.max(np.abs(got[..., 0] - h)) < (1e-9 if dt == "f64" else 1e-4)
    assert np.max(np.abs(got[..., 1])) < (1e-9 if dt == "f64" else 1e-4)
    before = md.clone()
    ctx.minimize_step(md)
    assert ctx.minimize_state()[0] == nit and torch.equal(md, before)


def test_minimize_is_deterministic_and_graph_capturable():
    """Repeated runs are bit-identical (fixed-order sums), and one captured iteration, replayed,
    follows the eager iterations: no host round trip inside an iteration."""
    n, d = (64, 32, 4), (3e-9, 3e-9, 3e-9)
    cfg = cfg_for(n, d, terms=1 | 2)
    m0 = torch.from_numpy(w.box_filter_renormalise(w.random_unit_vectors(9, n)).astype(np.float32))
    runs = []
    for use_graph in (False, False, True):
        ctx = make_ctx(cfg, "f32")
        ctx.minimize_init(2e-7, 1e-10, 1e-4, 0.0)
        mm = m0.cuda()
        if use_graph:
            s = torch.cuda.Stream()
            s.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(s):
                ctx.use_current_stream()
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=s):
                    ctx.minimize_step(mm)
                for _ in range(8):          # the capture itself enqueued nothing
                    g.replay()
            s.synchronize()
        else:
            for _ in range(8):
                ctx.minimize_step(mm)
        st = ctx.minimize_state()
        runs.append((mm.cpu().clone(), st))
        ctx.close()
    assert torch.equal(runs[0][0], runs[1][0]) and runs[0][1] == runs[1][1]
    assert torch.equal(runs[0][0], runs[2][0]) and runs[2][1][0] == 8 and runs[0][1] == runs[2][1]

"""Per-cell Ms and A (reading Q31) through the C ABI against the oracle's O14:
fields term by term, H_eff, dm/dt, RK4 / RKF45 / minimiser steps with vacuum cells."""
import numpy as np
import pytest
import torch

import workloads as w
from gpu_util import TOL, TRAJ_TOL, make_ctx, np_dtype, round_input, to_dev

pytestmark = pytest.mark.gpu


def cfg_for(n, d, **kw):
    base = w.get_config(1)
    return w.Config(**{**base.__dict__, "n": n, "d": d, "name": "t", **kw})


def material(n, seed, vacuum=True):
    rng = np.random.default_rng(seed)
    Ms = rng.uniform(3e5, 1e6, n)
    A = rng.uniform(0.5e-11, 2e-11, n)
    if vacuum:
        Ms[n[0] // 2:, : max(1, n[1] // 3)] = 0.0        # a notch of vacuum
        A[Ms == 0.0] = 0.0
        A[0, -1] = 0.0                                   # decoupled magnetic cells
    return Ms, A


def setup(oracle, cfg, dt, Ms, A, extra=None):
    kw = dict(n=cfg.n, d=cfg.d, Ms=cfg.Ms, Aex=cfg.Aex, Ku=cfg.Ku, axis=cfg.axis, alpha=cfg.alpha, gamma=cfg.gamma,
              Hext=cfg.Hext, terms=cfg.terms, **(extra or {}))
    Msr, Ar = Ms.astype(np_dtype(dt)), A.astype(np_dtype(dt))       # both sides see the rounded parameters
    P = oracle.Problem(Ms_cells=Msr.astype(np.float64), A_cells=Ar.astype(np.float64), **kw).prepare()
    ctx = make_ctx(cfg, dt)
    ctx.set_material_cells(to_dev(Msr), to_dev(Ar))
    return P, ctx


@pytest.mark.parametrize("dt", ["f64", "f32"])
@pytest.mark.parametrize("n,d", [((16, 16, 2), (5e-9, 5e-9, 3e-9)), ((12, 10, 6), (2e-9, 2e-9, 2e-9)),
                                 ((32, 16, 8), (4e-9, 3e-9, 2e-9)), ((9, 5, 1), (2e-9, 3e-9, 4e-9)),
                                 ((64, 64, 64), (3e-9, 3e-9, 3e-9))])
def test_terms_heff_and_rhs(oracle, n, d, dt):
    terms = 1 | 2 | 4 | 8 | 16 | 32
    cfg = cfg_for(n, d, Ku=4e5, axis=(0.0, 0.6, 0.8), alpha=0.3, Hext=(1e4, -2e4, 3e4), terms=terms)
    Ms, A = material(n, 11)
    extra = dict(D=2.5e-3, edmi=oracle.DMI_INTERFACIAL, stt_p=(0.0, 0.6, 0.8), stt_damp=4e3, stt_field=1.5e3)
    P, ctx = setup(oracle, cfg, dt, Ms, A, extra)
    ctx.set_dmi(2.5e-3)
    ctx.set_stt((0.0, 0.6, 0.8), 4e3, 1.5e3)
    m0 = w.random_unit_vectors(808, n)
    m0[Ms == 0.0] = 0.0
    m, m64 = round_input(m0, dt)
    md = to_dev(m)

    def only(t):
        Q = oracle.Problem(**{**P.__dict__, "terms": t})
        return Q.heff(m64)
    for name, got, ref in (("demag", ctx.demag_field(md), only(1)), ("exchange", ctx.exchange_field(md), only(2)),
                           ("dmi", ctx.dmi_field(md), only(16)), ("heff", ctx.heff(md), P.heff(m64)),
                           ("rhs", ctx.llg_rhs(md), P.llg_rhs(m64))):
        l2, mx = w.field_errors(got.cpu().numpy(), ref)
        assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (name, l2, mx)
    k = ctx.llg_rhs(md).cpu().numpy()
    assert np.all(k[Ms == 0.0] == 0.0)


@pytest.mark.parametrize("dt", ["f64", "f32"])
def test_rk4_rkf45_and_minimiser_with_vacuum(oracle, dt):
    n, d = (24, 12, 2), (4e-9, 4e-9, 3e-9)
    cfg = cfg_for(n, d, alpha=0.5, terms=1 | 2 | 8, Hext=(2e4, 1e4, 0.0))
    Ms, A = material(n, 12)
    P, ctx = setup(oracle, cfg, dt, Ms, A)
    m0 = w.box_filter_renormalise(w.random_unit_vectors(909, n))
    m0[Ms == 0.0] = 0.0
    m, m64 = round_input(m0, dt)
    md, ref = to_dev(m), m64.copy()
    for _ in range(10):
        ctx.rk_step(md, cfg.dt)
        ref = P.rk4_step(ref, cfg.dt)
        assert w.traj_error(md.cpu().numpy(), ref) <= TRAJ_TOL[dt]
    got = md.cpu().numpy()
    assert np.all(got[Ms == 0.0] == 0.0) and np.all(np.isfinite(got))
    ctx.rkf45_init(dt0=1e-13, tol=1e-6)
    for _ in range(4):
        st = ctx.rkf45_state()
        ref, err, acc, dtn = P.rkf45_step(ref, st["dt_next"], 1e-6)
        ctx.rkf45_step(md)
        assert w.traj_error(md.cpu().numpy(), ref) <= TRAJ_TOL[dt]
    bb = oracle.BBMinimizer(P, ref, tau0=2e-7, tau_min=1e-10, tau_max=1e-4, tol=1e-9)
    ctx.minimize_init(2e-7, 1e-10, 1e-4, 1e-9)
    if dt == "f32":
        bb.m = md.cpu().numpy().astype(np.float64)       # restart both sides from the same fp32 state
    else:
        md.copy_(to_dev(bb.m))
    for _ in range(10):
        bb.step()
        ctx.minimize_step(md)
        assert w.traj_error(md.cpu().numpy(), bb.m) <= TRAJ_TOL[dt]
    assert torch.isfinite(md).all() and np.all(md.cpu().numpy()[Ms == 0.0] == 0.0)


def test_cells_can_be_cleared_again(oracle):
    n, d = (16, 8, 4), (2e-9, 2e-9, 2e-9)
    cfg = cfg_for(n, d)
    Ms, A = material(n, 13, vacuum=False)
    P, ctx = setup(oracle, cfg, "f64", Ms, A)
    m = w.random_unit_vectors(1, n)
    ctx.set_material_cells(None, None)
    from gpu_util import make_problem
    ref = make_problem(oracle, cfg).heff(m)
    l2, mx = w.field_errors(ctx.heff(to_dev(m)).cpu().numpy(), ref)
    assert l2 <= TOL["f64"]


@pytest.mark.parametrize("dt", ["f64", "f32"])
def test_uniform_A_vacuum_neighbour_is_no_exchange_partner(oracle, dt):
    """Ms_cells with zeros, A_cells = NULL (uniform A), arbitrary non-zero vectors stored in the vacuum cells:
    the exchange field of the magnet does not see them (reading Q31: vacuum interface = mesh boundary)."""
    n, d = (16, 12, 4), (3e-9, 3e-9, 2e-9)
    cfg = cfg_for(n, d, terms=2)
    Ms = np.full(n, 8e5)
    Ms[8:] = 0.0
    m, m64 = round_input(w.random_unit_vectors(909, n), dt)          # vacuum cells hold unit vectors too
    Msr = Ms.astype(np_dtype(dt))
    P = oracle.Problem(n=n, d=d, Ms=cfg.Ms, Aex=cfg.Aex, terms=2, Ms_cells=Msr.astype(np.float64))
    ctx = make_ctx(cfg, dt)
    ctx.set_material_cells(to_dev(Msr), None)
    for got in (ctx.exchange_field(to_dev(m)), ctx.heff(to_dev(m))):
        got = got.cpu().numpy()
        l2, mx = w.field_errors(got, P.heff(m64))
        assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (l2, mx)
        ref_magnet = oracle.exchange(d, cfg.Ms, cfg.Aex, m64[:8])    # the magnet alone, Neumann at x = 7
        l2, mx = w.field_errors(got[:8], ref_magnet)
        assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (l2, mx)
        assert np.all(got[8:] == 0.0)
    ctx.close()

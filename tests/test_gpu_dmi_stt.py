"""DMI (eq. 3) and the spin-torque field in the fused pointwise pass,
against the oracle's O11 / O12, element by element, through the C ABI."""
import numpy as np
import pytest

import workloads as w
from gpu_util import TOL, TRAJ_TOL, make_ctx, make_problem, round_input, to_dev

pytestmark = pytest.mark.gpu

MESHES = [((16, 16, 2), (5e-9, 5e-9, 3e-9)), ((8, 4, 1), (3e-9, 4e-9, 5e-9)), ((1, 1, 4), (1e-9, 2e-9, 3e-9)),
          ((32, 16, 8), (4e-9, 3e-9, 2e-9)), ((9, 15, 5), (2e-9, 3e-9, 4e-9)), ((64, 32, 16), (2e-9, 2e-9, 2e-9)),
          ((12, 10, 6), (2e-9, 2e-9, 2e-9)), ((1, 1, 1), (1e-9, 1e-9, 1e-9))]


def cfg_for(n, d, **kw):
    base = w.get_config(1)
    return w.Config(**{**base.__dict__, "n": n, "d": d, "name": "t", **kw})


@pytest.mark.parametrize("dt", ["f64", "f32"])
@pytest.mark.parametrize("kind", ["interfacial", "bulk", "general"])
@pytest.mark.parametrize("n,d", MESHES)
def test_dmi_field(oracle, n, d, kind, dt):
    cfg = cfg_for(n, d)
    e = {"interfacial": oracle.DMI_INTERFACIAL, "bulk": oracle.DMI_BULK,
         "general": ((0.3, -1.0, 0.5), (0.7, 0.2, -0.4), (-0.6, 0.1, 0.9))}[kind]
    D = 3.0e-3
    m, m64 = round_input(w.random_unit_vectors(404, n), dt)
    ref = oracle.dmi(d, cfg.Ms, D, e, m64)
    ctx = make_ctx(cfg, dt, terms=16)
    ctx.set_dmi(D, e)
    got = ctx.dmi_field(to_dev(m)).cpu().numpy()
    if np.max(np.abs(ref)) == 0.0:
        assert np.all(got == 0.0)
        return
    l2, mx = w.field_errors(got, ref)
    assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (l2, mx)


@pytest.mark.parametrize("dt", ["f64", "f32"])
@pytest.mark.parametrize("n,d", [((16, 16, 2), (5e-9, 5e-9, 3e-9)), ((30, 20, 1), (2e-9, 2e-9, 1e-9)),
                                 ((32, 16, 8), (4e-9, 3e-9, 2e-9))])
def test_all_terms_heff_rhs_and_rk4(oracle, n, d, dt):
    """demag + exchange + anisotropy + Zeeman + DMI + spin-torque field: H_eff, dm/dt, 10 RK4 steps."""
    terms = 1 | 2 | 4 | 8 | 16 | 32
    cfg = cfg_for(n, d, Ku=4e5, axis=(0.0, 0.6, 0.8), alpha=0.3, Hext=(1e4, -2e4, 3e4), terms=terms)
    D, p, ad, af = 2.5e-3, (0.0, 0.6, 0.8), 4.0e3, 1.5e3
    m, m64 = round_input(w.random_unit_vectors(505, n), dt)
    P = make_problem(oracle, cfg)
    P.D, P.edmi, P.stt_p, P.stt_damp, P.stt_field = D, oracle.DMI_INTERFACIAL, p, ad, af
    ctx = make_ctx(cfg, dt)
    ctx.set_dmi(D)
    ctx.set_stt(p, ad, af)
    md = to_dev(m)
    for name, got, ref in (("heff", ctx.heff(md), P.heff(m64)), ("rhs", ctx.llg_rhs(md), P.llg_rhs(m64))):
        l2, mx = w.field_errors(got.cpu().numpy(), ref)
        assert l2 <= TOL[dt], (name, l2, mx)
    mo = m64.copy()
    for _ in range(10):
        ctx.rk_step(md, cfg.dt)
        mo = P.rk4_step(mo, cfg.dt)
        assert w.traj_error(md.cpu().numpy(), mo) <= TRAJ_TOL[dt]


@pytest.mark.parametrize("dt", ["f64", "f32"])
def test_stt_field_alone(oracle, dt):
    n, d = (16, 8, 4), (2e-9, 2e-9, 2e-9)
    cfg = cfg_for(n, d, terms=32)
    m, m64 = round_input(w.random_unit_vectors(606, n), dt)
    ctx = make_ctx(cfg, dt)
    ctx.set_stt((1.0, 2.0, 2.0), 7.0e3, -3.0e3)       # normalised by the library
    ref = oracle.stt(np.array([1.0, 2.0, 2.0]) / 3.0, 7.0e3, -3.0e3, m64)
    l2, mx = w.field_errors(ctx.heff(to_dev(m)).cpu().numpy(), ref)
    assert l2 <= TOL[dt], (l2, mx)

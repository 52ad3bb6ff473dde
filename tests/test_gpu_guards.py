"""Out-of-bounds writes: every output of the field and step calls sits between guard bands of a fixed bit
pattern that must come back untouched, over meshes that reach every demag path (x-first kernels with partial
tiles along every axis, TMA box stores, the z tile pass, L = 1024, embedded, generic, slab layout)."""
import numpy as np
import pytest
import torch

import workloads as w
from gpu_util import make_ctx, np_dtype, torch_dtype

pytestmark = pytest.mark.gpu

GUARD = 4096   # elements on each side
CASES = [((64, 64, 16), 0), ((100, 64, 18), 0), ((64, 128, 30), 0), ((128, 100, 54), 0), ((64, 64, 350), 0),
         ((1024, 64, 18), 0), ((64, 1024, 18), 0), ((64, 64, 16), 3), ((12, 10, 3), 0), ((60, 50, 20), 0), ((16, 16, 2), 0)]


def guarded(n, dt, fill=None):
    size = int(np.prod(n)) * 3
    buf = torch.full((size + 2 * GUARD,), -7.25, dtype=torch_dtype(dt), device="cuda")
    view = buf[GUARD:GUARD + size].view(*n, 3)
    assert view.data_ptr() % 16 == 0
    if fill is not None:
        view.copy_(fill)
    return buf, view


def guards_intact(buf):
    return bool((buf[:GUARD] == -7.25).all()) and bool((buf[-GUARD:] == -7.25).all())


@pytest.mark.parametrize("dt", ["f32", "f64"])
@pytest.mark.parametrize("n,slabs", CASES)
def test_outputs_stay_inside_their_buffers(n, slabs, dt):
    base = w.get_config(1)
    cfg = w.Config(**{**base.__dict__, "n": n, "d": (4e-9, 3e-9, 2e-9), "name": "g", "terms": 1 | 2 | 8,
                      "Hext": (1e4, -2e4, 3e4)})
    ctx = make_ctx(cfg, dt, slabs=slabs)
    m = torch.from_numpy(w.random_unit_vectors(31, n).astype(np_dtype(dt))).cuda()
    mb, mv = guarded(n, dt, m)
    for call in (ctx.demag_field, ctx.exchange_field, ctx.heff, ctx.llg_rhs):
        ob, ov = guarded(n, dt)
        call(mv, ov)
        torch.cuda.synchronize()
        assert guards_intact(ob), (call.__name__, n, dt)
        assert bool(torch.isfinite(ov).all()) and not bool((ov == -7.25).all())
        assert guards_intact(mb) and torch.equal(mv, m), ("input changed", call.__name__)
    ctx.rk_step(mv, 1e-13)
    ctx.rk_steps(mv, 1e-13, 2)
    torch.cuda.synchronize()
    assert guards_intact(mb)
    assert bool(torch.isfinite(mv).all())
    ctx.close()


@pytest.mark.parametrize("dt", ["f32", "f64"])
@pytest.mark.parametrize("n,slabs", CASES)
def test_workspaces_are_not_overrun(n, slabs, dt):
    """The library carves the two caller-owned workspaces itself (mm_ctx_workspace_bytes): exactly that many bytes
    between guard bands, S0 (mm_demag_init), the field calls, RK4, one RKF45 attempt and one minimiser iteration."""
    from paper_2606_01114_b200 import Context
    base = w.get_config(1)
    cfg = w.Config(**{**base.__dict__, "n": n, "d": (4e-9, 3e-9, 2e-9), "name": "g", "terms": 1 | 2 | 8,
                      "Hext": (1e4, -2e4, 3e4)})
    ctx = Context(cfg.n, cfg.d, dtype=torch_dtype(dt), allocate=False, slabs=slabs)
    p, s = ctx.workspace_bytes()
    G = 65536
    pers = torch.full((p + 2 * G,), 0x5A, dtype=torch.uint8, device="cuda")
    scr = torch.full((s + 2 * G,), 0x5A, dtype=torch.uint8, device="cuda")
    assert pers.data_ptr() % 256 == 0 and scr.data_ptr() % 256 == 0
    ctx._ws = (pers, scr)
    ctx._call("mm_ctx_set_workspace", pers.data_ptr() + G, p, scr.data_ptr() + G, s)
    ctx.use_current_stream()
    ctx.set_material(cfg.Ms, cfg.Aex, cfg.Ku, cfg.axis, cfg.alpha, cfg.gamma)
    ctx.set_zeeman(cfg.Hext)
    ctx.set_terms(cfg.terms)
    ctx.demag_init()
    m = torch.from_numpy(w.random_unit_vectors(32, n).astype(np_dtype(dt))).cuda()
    out = torch.empty_like(m)
    ctx.demag_field(m, out)
    ctx.llg_rhs(m, out)
    ctx.rk_step(m, 1e-13)
    ctx.rkf45_init(0.0, 1e-13, 1e-6, 1e-16, 1e-11)
    ctx.rkf45_step(m)
    ctx.minimize_init(1e-6, 1e-10, 1e-3, 1e-9)
    ctx.minimize_step(m)
    torch.cuda.synchronize()
    for name, buf in (("persistent", pers), ("scratch", scr)):
        assert bool((buf[:G] == 0x5A).all()) and bool((buf[-G:] == 0x5A).all()), (name, n, dt)
    assert bool(torch.isfinite(m).all())
    ctx.close()

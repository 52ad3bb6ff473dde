"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

The oracle cannot run a dense 33.5 M-cell direct sum, so full-size checks use
 (1) sparse sources: a handful of magnetised cells, every sampled output is
     -Ms sum_s N(i - j_s) m_s with N from the oracle's literal quad-precision definition;
 (2) invariants that hold at any size: the trace rule on the three uniform states
     (sum_d -H_d.e_d / Ms = 1 at EVERY cell) and linearity on dense random input;
 (3) config 3 (256x256x64, smoothed field, anisotropy) densely against the oracle FFT path.
"""
import numpy as np
import pytest
import torch

import workloads as w
from gpu_util import TOL, make_ctx, make_problem, round_input, to_dev

pytestmark = pytest.mark.gpu


def sparse_reference(oracle, cfg, ids, vecs, cells):
    nx, ny, nz = cfg.n
    ref = np.zeros((len(cells), 3))
    for a, cell in enumerate(cells):
        ci = np.array([cell // (ny * nz), (cell // nz) % ny, cell % nz])
        for sid, v in zip(ids, vecs):
            si = np.array([sid // (ny * nz), (sid // nz) % ny, sid % nz])
            off = ci - si
            Np = oracle.newell_point(cfg.d, int(off[0]), int(off[1]), int(off[2]))
            full = np.array([[Np[0], Np[3], Np[4]], [Np[3], Np[1], Np[5]], [Np[4], Np[5], Np[2]]])
            ref[a] += -cfg.Ms * full @ v
    return ref


@pytest.mark.parametrize("cfg_id,dt", [(4, "f32"), (4, "f64"), (3, "f32")])
def test_sparse_sources_fullsize(oracle, cfg_id, dt):
    cfg = w.get_config(cfg_id)
    m64, ids = w.sparse_sources(cfg.seed, cfg.n, 6)
    m, mref = round_input(m64, dt)
    cells = np.unique(np.concatenate([w.sample_cells(cfg.seed, cfg.n, 150), ids]))
    ref = sparse_reference(oracle, cfg, ids, mref.reshape(-1, 3)[ids], cells)
    ctx = make_ctx(cfg, dt, terms=1)
    got = ctx.demag_field(to_dev(m)).cpu().numpy().reshape(-1, 3)[cells]
    l2, mx = w.field_errors(got, ref)
    assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (l2, mx)
    # far field individually: every sampled value is right to a relative accuracy set by the
    # absolute tolerance (fp64: far values ~1e-9 Ms still carry 3 digits)
    scale = np.max(np.abs(ref))
    assert np.all(np.abs(got - ref) <= 10 * TOL[dt] * scale)
    ctx.close()


@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_trace_rule_and_linearity_config4(dt):
    cfg = w.get_config(4)
    ctx = make_ctx(cfg, dt, terms=1)
    tdt = torch.float32 if dt == "f32" else torch.float64
    tot = torch.zeros(cfg.n, dtype=torch.float64, device="cuda")
    m = torch.zeros(cfg.n + (3,), dtype=tdt, device="cuda")
    H = torch.empty_like(m)
    for c in range(3):
        m.zero_()
        m[..., c] = 1.0
        ctx.demag_field(m, H)
        tot -= H[..., c].double() / cfg.Ms
    err = float((tot - 1.0).abs().max())
    assert err <= (1e-11 if dt == "f64" else 2e-5), err
    # linearity on dense random input (bench.py's input)
    g = torch.Generator(device="cuda")
    g.manual_seed(11)
    a = torch.randn(cfg.n + (3,), dtype=tdt, device="cuda", generator=g)
    a /= a.norm(dim=-1, keepdim=True)
    b = torch.randn(cfg.n + (3,), dtype=tdt, device="cuda", generator=g)
    b /= b.norm(dim=-1, keepdim=True)
    Ha = ctx.demag_field(a).double()
    Hb = ctx.demag_field(b).double()
    Hab = ctx.demag_field((a + 0.5 * b).contiguous()).double()
    d = float((Hab - (Ha + 0.5 * Hb)).abs().max() / Ha.abs().max())
    assert d <= (1e-12 if dt == "f64" else 2e-5), d
    ctx.close()


def test_config3_dense_heff_and_rhs(oracle):
    """Config 3: 256x256x64, fp32, smoothed random field, demag + exchange + anisotropy."""
    cfg = w.get_config(3)
    m, mref = round_input(cfg.initial_m(), "f32")
    P = make_problem(oracle, cfg)
    ctx = make_ctx(cfg, "f32")
    md = to_dev(m)
    l2, mx = w.field_errors(ctx.demag_field(md).cpu().numpy(), oracle.demag_fft(P.Nhat, cfg.Ms, mref))
    assert l2 <= TOL["f32"], ("demag", l2, mx)
    l2, mx = w.field_errors(ctx.heff(md).cpu().numpy(), P.heff(mref))
    assert l2 <= TOL["f32"], ("heff", l2, mx)
    l2, mx = w.field_errors(ctx.llg_rhs(md).cpu().numpy(), P.llg_rhs(mref))
    assert l2 <= TOL["f32"], ("rhs", l2, mx)
    # sampled direct sum (no FFT on the reference side at all)
    cells = w.sample_cells(cfg.seed, cfg.n, 40)
    ref = oracle.demag_direct_sampled(P.N, cfg.Ms, mref, cells)
    got = ctx.demag_field(md).cpu().numpy().reshape(-1, 3)[cells]
    l2, mx = w.field_errors(got, ref)
    assert l2 <= TOL["f32"], ("sampled", l2, mx)
    ctx.close()


@pytest.mark.parametrize("dt", ["f32", "f64"])
@pytest.mark.parametrize("n", w.SWEEP_MESHES)
def test_sweep_meshes_sparse(oracle, n, dt):
    """Config 5: every sweep size (64^3 ... 1024 x 1024 x 128, incl. the 1024-point axes), fp32 and
    fp64: sparse-source parity against the oracle's literal Newell definition."""
    cfg = w.get_config(5).with_mesh(n)
    m64, ids = w.sparse_sources(cfg.seed, cfg.n, 4)
    m, mref = round_input(m64, dt)
    cells = np.unique(np.concatenate([w.sample_cells(cfg.seed, cfg.n, 60), ids]))
    ref = sparse_reference(oracle, cfg, ids, mref.reshape(-1, 3)[ids], cells)
    ctx = make_ctx(cfg, dt, terms=1)
    assert ctx.path_name == "fast"
    md = to_dev(m)
    del m, mref, m64
    got = ctx.demag_field(md).reshape(-1, 3)[to_dev(cells)].cpu().numpy()
    l2, mx = w.field_errors(got, ref)
    assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (l2, mx)
    ctx.close()
    del ctx, md
    torch.cuda.empty_cache()

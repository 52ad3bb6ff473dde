"""Meshes whose sides are not powers of two: the paper's own workloads are
100 x 25 x 1, N = 100, 350, 400 cubes and 512 x 512 x 90
(PAPER.md:250).  The CUDA path pads to exactly 2n; references are the direct sum (O3), the oracle
FFT path at its own power-of-two period (reading Q27) and, at full size, sparse sources and the
trace rule.  The cubes and the multilayer run the two-register-stage x-first kernels
(demag_fast2.cu, demag_ztile.cu), everything else the generic run-time radix stages."""
import numpy as np
import pytest
import torch

import workloads as w
from gpu_util import TOL, TRAJ_TOL, make_ctx, make_problem, round_input, to_dev
from test_gpu_fullsize import sparse_reference

pytestmark = pytest.mark.gpu

SMALL = [((6, 5, 3), (3e-9, 4e-9, 5e-9)), ((7, 3, 2), (2e-9, 2e-9, 1e-9)), ((3, 1, 1), (1e-9, 2e-9, 3e-9)),
         ((12, 10, 1), (5e-9, 5e-9, 3e-9)), ((9, 15, 5), (2e-9, 3e-9, 4e-9)), ((25, 14, 6), (4e-9, 3e-9, 2e-9)),
         ((1, 21, 10), (1e-9, 2e-9, 3e-9)), ((49, 2, 27), (2e-9, 2e-9, 2e-9))]


def cfg_for(n, d, **kw):
    base = w.get_config(1)
    return w.Config(**{**base.__dict__, "n": n, "d": d, "name": "t", **kw})


def mirrored_nhat(oracle, n, d):
    """Real part of numpy's FFT of the oracle's Newell table mirrored onto the period-2n grid
    (offset -i at index 2n - i, index n zero: readings Q10, Q11), octant k <= n."""
    N = oracle.newell_octant(n, d)
    P = [oracle.padded(v) for v in n]
    parity = {0: (0, 0, 0), 1: (0, 0, 0), 2: (0, 0, 0), 3: (1, 1, 0), 4: (1, 0, 1), 5: (0, 1, 1)}
    out = []
    for comp in range(6):
        full = np.zeros(P)
        for sx in (0, 1):
            for sy in (0, 1):
                for sz in (0, 1):
                    sgn = (-1) ** (sx * parity[comp][0] + sy * parity[comp][1] + sz * parity[comp][2])
                    src = N[comp]
                    ix = np.arange(n[0]) if not sx else (P[0] - np.arange(n[0])) % P[0]
                    iy = np.arange(n[1]) if not sy else (P[1] - np.arange(n[1])) % P[1]
                    iz = np.arange(n[2]) if not sz else (P[2] - np.arange(n[2])) % P[2]
                    full[np.ix_(ix, iy, iz)] = sgn * src
        # offset 0 along a mirrored odd axis: N is structurally zero there, so the last write wins harmlessly
        F = np.fft.fftn(full)
        assert np.max(np.abs(F.imag)) < 1e-12
        o = tuple(1 if v == 1 else v + 1 for v in n)
        out.append(F.real[:o[0], :o[1], :o[2]])
    return np.stack(out)


@pytest.mark.parametrize("dt", ["f64", "f32"])
@pytest.mark.parametrize("n,d", SMALL)
def test_nhat_matches_fft_of_mirrored_table(oracle, n, d, dt):
    ctx = make_ctx(cfg_for(n, d), dt)
    got = ctx.nhat_export().cpu().numpy().astype(np.float64)
    ref = mirrored_nhat(oracle, n, d)
    assert np.max(np.abs(got - ref)) < (5e-14 if dt == "f64" else 2e-7)


@pytest.mark.parametrize("dt", ["f64", "f32"])
@pytest.mark.parametrize("n,d", SMALL + [((100, 25, 1), (5e-9, 5e-9, 3e-9))])
def test_demag_vs_direct_sum(oracle, n, d, dt):
    cfg = cfg_for(n, d)
    m, m64 = round_input(w.random_unit_vectors(111, n), dt)
    ref = oracle.demag_direct(oracle.newell_octant(n, d), cfg.Ms, m64)
    ctx = make_ctx(cfg, dt)
    got = ctx.demag_field(to_dev(m)).cpu().numpy()
    l2, mx = w.field_errors(got, ref)
    assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (l2, mx)


@pytest.mark.parametrize("dt", ["f64", "f32"])
@pytest.mark.parametrize("n", [(100, 50, 30), (90, 70, 18), (35, 120, 45), (200, 6, 14)])
def test_demag_vs_oracle_fft_medium(oracle, n, dt):
    """Several tiles per pass; reference = the oracle FFT path (period: next power of two)."""
    cfg = cfg_for(n, (4e-9, 3e-9, 2e-9))
    m, m64 = round_input(w.random_unit_vectors(212, n), dt)
    P = make_problem(oracle, cfg, terms=1)
    ref = oracle.demag_fft(P.Nhat, cfg.Ms, m64)
    ctx = make_ctx(cfg, dt)
    got = ctx.demag_field(to_dev(m)).cpu().numpy()
    l2, mx = w.field_errors(got, ref)
    assert l2 <= TOL[dt], (l2, mx)
    assert np.array_equal(got, ctx.demag_field(to_dev(m)).cpu().numpy())   # deterministic


@pytest.mark.parametrize("dt", ["f64", "f32"])
def test_sp4_grid_heff_rhs_and_rk4(oracle, dt):
    """The paper's SP4 mesh as published: 100 x 25 x 1 cells of 5 x 5 x 3 nm,
    Ms 8e5, A 1.3e-11, alpha 0.02, field (-24.6, 4.3, 0) mT: H_eff, dm/dt and 20 RK4 steps."""
    c2 = w.get_config(2)
    cfg = w.Config(**{**c2.__dict__, "n": (100, 25, 1), "d": (5e-9, 5e-9, 3e-9), "name": "sp4_as_published"})
    m, m64 = round_input(cfg.initial_m(), dt)
    P = make_problem(oracle, cfg)
    ctx = make_ctx(cfg, dt)
    md = to_dev(m)
    for name, got, ref in (("heff", ctx.heff(md), P.heff(m64)), ("rhs", ctx.llg_rhs(md), P.llg_rhs(m64))):
        l2, mx = w.field_errors(got.cpu().numpy(), ref)
        assert l2 <= TOL[dt], (name, l2, mx)
    mo = m64.copy()
    for _ in range(20):
        ctx.rk_step(md, cfg.dt)
        mo = P.rk4_step(mo, cfg.dt)
        assert w.traj_error(md.cpu().numpy(), mo) <= TRAJ_TOL[dt]


@pytest.mark.parametrize("n,dt", [((350, 350, 350), "f64"), ((100, 100, 100), "f64"), ((400, 400, 400), "f32"),
                                  ((512, 512, 90), "f32")])
def test_paper_meshes_fullsize(oracle, n, dt):
    """The paper's benchmark meshes at full size: sparse sources against the oracle's literal
    Newell values, and the trace rule at every cell."""
    cfg = w.get_config(5).with_mesh(n)
    m64, ids = w.sparse_sources(cfg.seed, cfg.n, 4)
    m, mref = round_input(m64, dt)
    cells = np.unique(np.concatenate([w.sample_cells(cfg.seed, cfg.n, 60), ids]))
    ref = sparse_reference(oracle, cfg, ids, mref.reshape(-1, 3)[ids], cells)
    ctx = make_ctx(cfg, dt, terms=1)
    got = ctx.demag_field(to_dev(m)).cpu().numpy().reshape(-1, 3)[cells]
    l2, mx = w.field_errors(got, ref)
    assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (l2, mx)
    tdt = torch.float32 if dt == "f32" else torch.float64
    tot = torch.zeros(cfg.n, dtype=torch.float64, device="cuda")
    mu = torch.zeros(cfg.n + (3,), dtype=tdt, device="cuda")
    H = torch.empty_like(mu)
    for c in range(3):
        mu.zero_()
        mu[..., c] = 1.0
        ctx.demag_field(mu, H)
        tot -= H[..., c].double() / cfg.Ms
    err = float((tot - 1.0).abs().max())
    assert err <= (1e-11 if dt == "f64" else 2e-5), err
    ctx.close()


@pytest.mark.parametrize("dt", ["f64", "f32"])
@pytest.mark.parametrize("n", [(16, 16, 2), (32, 16, 8), (64, 64, 64), (128, 64, 32), (25, 14, 6), (10, 6, 90),
                               (2, 2, 2), (70, 3, 4)])
def test_mixed_radix_xfirst_kernels_explicitly(oracle, n, dt):
    """path = 3 forces demag_mixed.cu (also on power-of-two meshes): N-hat export, field vs the oracle
    FFT path, agreement with the generic z-first passes, determinism."""
    cfg = cfg_for(n, (4e-9, 3e-9, 2e-9))
    m, m64 = round_input(w.random_unit_vectors(313, n), dt)
    P = make_problem(oracle, cfg, terms=1)
    ref = oracle.demag_fft(P.Nhat, cfg.Ms, m64)
    ctx = make_ctx(cfg, dt, terms=1, path=3)
    assert ctx.path_name == "mixed"
    got = ctx.demag_field(to_dev(m)).cpu().numpy()
    l2, mx = w.field_errors(got, ref)
    assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (l2, mx)
    assert np.array_equal(got, ctx.demag_field(to_dev(m)).cpu().numpy())
    nh = ctx.nhat_export().cpu().numpy().astype(np.float64)
    assert np.max(np.abs(nh - mirrored_nhat(oracle, n, cfg.d))) < (5e-14 if dt == "f64" else 2e-7)
    gen = make_ctx(cfg, dt, terms=1, path=1)
    assert gen.path_name == "generic"
    l2, mx = w.field_errors(gen.demag_field(to_dev(m)).cpu().numpy(), got)
    assert l2 <= TOL[dt], (l2, mx)


def test_mixed_radix_selection():
    from paper_2606_01114_b200 import MMError
    # the paper's own meshes run the x-first register-stage kernels (two-stage plans 700 = 28 x 25, 800 = 32 x 25,
    # 200 = 20 x 10; z below 256 layers at period 128, 256 or 512)
    for n in ((350, 350, 350), (400, 400, 400), (100, 100, 100), (512, 512, 90), (350, 64, 90), (128, 400, 100)):
        assert make_ctx(cfg_for(n, (4e-9,) * 3), "f64", terms=0).path_name == "fast", n
    assert make_ctx(cfg_for((350, 350, 350), (4e-9,) * 3), "f64", terms=0, path=3).path_name == "mixed"
    assert make_ctx(cfg_for((350, 350, 350), (4e-9,) * 3), "f64", terms=0, path=1).path_name == "generic"
    assert make_ctx(cfg_for((350, 350, 175), (4e-9,) * 3), "f64", terms=0).path_name == "fast"      # z at period 512
    assert make_ctx(cfg_for((350, 350, 300), (4e-9,) * 3), "f64", terms=0).path_name == "embedded"  # in 350^3
    assert make_ctx(cfg_for((350, 350, 8), (4e-9,) * 3), "f64", terms=0).path_name == "embedded"    # in 16 layers
    assert make_ctx(cfg_for((350, 350, 4), (4e-9,) * 3), "f64", terms=0).path_name == "generic"     # too thin
    assert make_ctx(cfg_for((512, 512, 128), (4e-9,) * 3), "f32", terms=0).path_name == "fast"
    assert make_ctx(cfg_for((100, 25, 1), (5e-9, 5e-9, 3e-9)), "f64", terms=0).path_name == "generic"
    assert make_ctx(cfg_for((9, 15, 5), (1e-9,) * 3), "f64", terms=0).path_name == "generic"   # ny 3 nz odd
    with pytest.raises(MMError):
        make_ctx(cfg_for((100, 25, 1), (5e-9, 5e-9, 3e-9)), "f64", terms=0, path=3)


@pytest.mark.parametrize("dt", ["f64", "f32"])
@pytest.mark.parametrize("n", [(60, 50, 40), (40, 64, 96), (96, 100, 80)])
def test_embedding_in_the_enclosing_mesh(oracle, n, dt):
    """Automatic selection places these meshes in the corner of 64^3 / 64 x 64 x 100 / 100 x 100 x 90, the
    smallest meshes the x-first kernels cover, and runs them there (cells outside carry no magnetisation):
    dense parity vs the oracle FFT path, agreement with the generic passes, H_eff + LLG through the cropped
    field, determinism."""
    cfg = cfg_for(n, (4e-9, 3e-9, 2e-9), terms=1 | 2 | 8, Hext=(1e4, 2e4, -3e4))
    m, m64 = round_input(w.random_unit_vectors(414, n), dt)
    P = make_problem(oracle, cfg)
    ctx = make_ctx(cfg, dt)
    assert ctx.path_name == "embedded"
    md = to_dev(m)
    got = ctx.demag_field(md).cpu().numpy()
    l2, mx = w.field_errors(got, oracle.demag_fft(P.Nhat, cfg.Ms, m64))
    assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (l2, mx)
    assert np.array_equal(got, ctx.demag_field(md).cpu().numpy())
    # the scratch workspace holds no state between calls (mm_b200.h): garbage in it changes nothing
    ctx._ws[1].fill_(0x7F)
    assert np.array_equal(got, ctx.demag_field(md).cpu().numpy())
    l2, mx = w.field_errors(ctx.llg_rhs(md).cpu().numpy(), P.llg_rhs(m64))
    assert l2 <= TOL[dt], (l2, mx)
    gen = make_ctx(cfg, dt, path=1)
    assert gen.path_name == "generic"
    l2, mx = w.field_errors(gen.demag_field(md).cpu().numpy(), got)
    assert l2 <= TOL[dt], (l2, mx)
    from paper_2606_01114_b200 import MMError
    with pytest.raises(MMError):
        ctx.nhat_export()


# every mixed-radix two-stage plan along each axis it serves, with dense input and several tiles per pass
PLAN_MESHES = [(100, 100, 100), (350, 64, 64), (64, 350, 64), (64, 64, 350), (400, 64, 90), (64, 400, 100),
               (64, 64, 400)]


@pytest.mark.slow
@pytest.mark.parametrize("n", PLAN_MESHES)
def test_register_stage_plans_dense_vs_oracle_fft(oracle, n):
    """700 = 28 x 25, 800 = 32 x 25, 200 = 20 x 10 along x, y and z and 180 = 20 x 9 along z: dense seeded input,
    fp32 and fp64, element by element against the oracle FFT path (its own power-of-two period, reading Q27);
    ragged last tiles (3 nz and ny 3 nz / 2 are not multiples of a tile row); agreement with the generic passes."""
    cfg = cfg_for(n, (4e-9, 3e-9, 2e-9))
    m32 = w.random_unit_vectors(515, n).astype(np.float32)
    m64 = m32.astype(np.float64)                      # one input for both dtypes
    P = make_problem(oracle, cfg, terms=1)
    ref = oracle.demag_fft(P.Nhat, cfg.Ms, m64)
    for dt in ("f32", "f64"):
        md = to_dev(m64.astype(np.float32 if dt == "f32" else np.float64))
        ctx = make_ctx(cfg, dt, terms=1)
        assert ctx.path_name == "fast"
        got = ctx.demag_field(md).cpu().numpy()
        l2, mx = w.field_errors(got, ref)
        assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (n, dt, l2, mx)
        assert np.array_equal(got, ctx.demag_field(md).cpu().numpy())
        ctx.close()
        if n[0] * n[1] * n[2] <= 1 << 21:
            gen = make_ctx(cfg, dt, terms=1, path=1)
            l2, mx = w.field_errors(gen.demag_field(md).cpu().numpy(), got)
            assert l2 <= TOL[dt], (n, dt, l2, mx)
            gen.close()


@pytest.mark.parametrize("dt", ["f64", "f32"])
def test_register_stage_plans_nhat_and_direct_sum(oracle, dt):
    """100 x 100 x 64 (plans 20 x 10 along x and y): the exported N-hat octant against numpy's FFT of the
    mirrored oracle table; 100 x 100 x 90 (z at period 256): the field against sampled direct sums O3 (no FFT
    on the reference side); its table is not exported at period 2 n."""
    from paper_2606_01114_b200 import MMError
    n0, d = (100, 100, 64), (5e-9, 4e-9, 3e-9)
    ctx = make_ctx(cfg_for(n0, d), dt, terms=1)
    assert ctx.path_name == "fast"
    nh = ctx.nhat_export().cpu().numpy().astype(np.float64)
    assert np.max(np.abs(nh - mirrored_nhat(oracle, n0, d))) < (5e-14 if dt == "f64" else 2e-7)
    ctx.close()
    n = (100, 100, 90)
    cfg = cfg_for(n, d)
    ctx = make_ctx(cfg, dt, terms=1)
    assert ctx.path_name == "fast"
    with pytest.raises(MMError):
        ctx.nhat_export()
    m, m64 = round_input(w.random_unit_vectors(616, n), dt)
    cells = w.sample_cells(17, n, 50)
    ref = oracle.demag_direct_sampled(oracle.newell_octant(n, d), cfg.Ms, m64, cells)
    got = ctx.demag_field(to_dev(m)).cpu().numpy().reshape(-1, 3)[cells]
    l2, mx = w.field_errors(got, ref)
    assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (l2, mx)
    ctx.close()

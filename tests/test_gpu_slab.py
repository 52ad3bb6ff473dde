"""Slab decomposition of the demag convolution ("sharded into contiguous slabs
along the x-axis", :47 "all-to-all transpose", :227), emulated on one device: R ranks, each owning an x slab of m
and H and a ky slab of the half spectrum and of the Fourier-space tensor; the forward y pass stores every
spectrum row into its owner's buffer and the inverse y pass gathers it back through a per-rank pointer table
(mm_ctx_set_slabs).  Parity against the oracle FFT path and agreement with the unsharded kernels."""
import numpy as np
import pytest

import workloads as w
from gpu_util import TOL, make_ctx, make_problem, np_dtype, to_dev

pytestmark = pytest.mark.gpu


def cfg_for(n, d=(4e-9, 3e-9, 2e-9), **kw):
    base = w.get_config(1)
    return w.Config(**{**base.__dict__, "n": n, "d": d, "name": "slab", **kw})


# even and uneven splits: 65 (101, 129) spectrum rows and 64 (100, 128) x planes over 2, 3, 4, 8 ranks; every K3 kernel
# (64-, 128- and 256-layer warp-per-pencil kernels incl. fewer layers than their capacity; the tile pass is covered below)
MESHES = [(64, 64, 64), (128, 64, 64), (64, 128, 128), (100, 100, 90), (64, 64, 200)]


@pytest.mark.parametrize("n", MESHES)
def test_slab_decomposition_matches_oracle_and_unsharded(oracle, n):
    cfg = cfg_for(n)
    m32 = w.random_unit_vectors(919, n).astype(np.float32)
    m64 = m32.astype(np.float64)
    P = make_problem(oracle, cfg, terms=1)
    ref = oracle.demag_fft(P.Nhat, cfg.Ms, m64)
    for dt in ("f32", "f64"):
        md = to_dev(m64.astype(np_dtype(dt)))
        whole = make_ctx(cfg, dt, terms=1)
        base = whole.demag_field(md).cpu().numpy()
        whole.close()
        for R in (1, 2, 3, 4, 8):
            ctx = make_ctx(cfg, dt, terms=1, slabs=R)
            got = ctx.demag_field(md).cpu().numpy()
            l2, mx = w.field_errors(got, ref)
            assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (n, dt, R, l2, mx)
            l2, mx = w.field_errors(got, base)
            assert l2 <= TOL[dt], (n, dt, R, l2, mx)           # same field as the unsharded kernels, to rounding
            assert np.array_equal(got, ctx.demag_field(md).cpu().numpy())
            ctx.close()


@pytest.mark.slow
@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_slab_decomposition_tile_pass_and_full_step(oracle, dt):
    """nz = 350 (the tile pass of demag_ztile.cu in the slab layout) and the whole H_eff + LLG right-hand side
    through a sharded demag field, R = 4."""
    n = (64, 64, 350)
    cfg = cfg_for(n, terms=1 | 2 | 8, Hext=(1e4, -2e4, 3e4))
    m32 = w.random_unit_vectors(929, n).astype(np.float32)
    m64 = m32.astype(np.float64)
    P = make_problem(oracle, cfg)
    ctx = make_ctx(cfg, dt, slabs=4)
    md = to_dev(m64.astype(np_dtype(dt)))
    l2, mx = w.field_errors(ctx.demag_field(md).cpu().numpy(), oracle.demag_fft(P.Nhat, cfg.Ms, m64))
    assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (l2, mx)
    l2, mx = w.field_errors(ctx.llg_rhs(md).cpu().numpy(), P.llg_rhs(m64))
    assert l2 <= TOL[dt], (l2, mx)
    ctx.close()


def test_slab_layout_needs_the_xfirst_kernels():
    from paper_2606_01114_b200 import MMError
    with pytest.raises(MMError) as ei:
        make_ctx(cfg_for((16, 16, 2)), "f64", terms=1, slabs=2)
    assert ei.value.status == 2
    with pytest.raises(MMError):
        make_ctx(cfg_for((64, 64, 64)), "f64", terms=1, slabs=9)

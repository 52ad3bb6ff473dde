"""The x-first fast demag kernels (demag_fast.cu, demag_fast2.cu; K1..K5) against the oracle and
against the generic z-first passes, through the C ABI: several tiles per pass, every supported
radix plan."""
import numpy as np
import pytest

import workloads as w
from gpu_util import TOL, make_ctx, make_problem, round_input, to_dev

pytestmark = pytest.mark.gpu

MESHES = [(64, 64, 64), (128, 64, 64), (64, 256, 128), (256, 128, 64), (64, 64, 128)]


def cfg_for(n, d=(4e-9, 3e-9, 2e-9)):
    base = w.get_config(1)
    return w.Config(**{**base.__dict__, "n": n, "d": d, "name": "t"})


@pytest.mark.parametrize("dt", ["f64", "f32"])
@pytest.mark.parametrize("n", MESHES)
def test_fast_demag_vs_oracle_fft(oracle, n, dt):
    cfg = cfg_for(n)
    m, m64 = round_input(w.random_unit_vectors(404, n), dt)
    P = make_problem(oracle, cfg, terms=1)
    ref = oracle.demag_fft(P.Nhat, cfg.Ms, m64)
    md = to_dev(m)
    ctx = make_ctx(cfg, dt, terms=1, path=2)
    assert ctx.path_name == "fast"
    got = ctx.demag_field(md).cpu().numpy()
    l2, mx = w.field_errors(got, ref)
    assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (l2, mx)
    assert np.array_equal(got, ctx.demag_field(md).cpu().numpy())      # deterministic
    ctx.close()
    # the generic passes agree with the fast kernels to rounding
    ctx = make_ctx(cfg, dt, terms=1, path=1)
    assert ctx.path_name == "generic"
    l2, mx = w.field_errors(ctx.demag_field(md).cpu().numpy(), got)
    assert l2 <= TOL[dt], (l2, mx)
    ctx.close()


@pytest.mark.parametrize("dt", ["f64", "f32"])
def test_fast_nhat_export(oracle, dt):
    n, d = (64, 64, 64), (4e-9, 3e-9, 2e-9)
    ctx = make_ctx(cfg_for(n, d), dt, terms=1, path=2)
    got = ctx.nhat_export().cpu().numpy().astype(np.float64)
    Nhat = oracle.demag_fft_nhat(oracle.newell_octant(n, d))
    ref = Nhat[:, :n[0] + 1, :n[1] + 1, :n[2] + 1]
    assert np.max(np.abs(got - ref)) < (5e-14 if dt == "f64" else 2e-7)


def test_fast_vs_direct_sum_sampled(oracle):
    """No FFT on the reference side: sampled O(n) direct sums on a 64x64x64 mesh, fp64."""
    n, d = (64, 64, 64), (5e-9, 5e-9, 3e-9)
    cfg = cfg_for(n, d)
    m, m64 = round_input(w.random_unit_vectors(505, n), "f64")
    N = oracle.newell_octant(n, d)
    cells = w.sample_cells(9, n, 60)
    ref = oracle.demag_direct_sampled(N, cfg.Ms, m64, cells)
    ctx = make_ctx(cfg, "f64", terms=1, path=2)
    got = ctx.demag_field(to_dev(m)).cpu().numpy().reshape(-1, 3)[cells]
    l2, mx = w.field_errors(got, ref)
    assert l2 <= TOL["f64"], (l2, mx)


@pytest.mark.parametrize("dt", ["f32", "f64"])
@pytest.mark.parametrize("n", [(64, 64, 256), (128, 64, 256)])
def test_fast_wide_pencil_nz256(oracle, n, dt):
    """nz = 256 (Pz = 512): the one-pencil-per-warp z kernel with the split second stage, fp32 and fp64;
    several planes and mirror pairs per warp."""
    cfg = cfg_for(n)
    m, m64 = round_input(w.random_unit_vectors(606, n), dt)
    P = make_problem(oracle, cfg, terms=1)
    ref = oracle.demag_fft(P.Nhat, cfg.Ms, m64)
    md = to_dev(m)
    ctx = make_ctx(cfg, dt, terms=1, path=2)
    assert ctx.path_name == "fast"
    got = ctx.demag_field(md).cpu().numpy()
    l2, mx = w.field_errors(got, ref)
    assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (l2, mx)
    assert np.array_equal(got, ctx.demag_field(md).cpu().numpy())
    ctx.close()


def test_fast_path_rejects_meshes_it_does_not_cover():
    """Fewer than 16 layers are served by the generic passes; requiring the x-first kernels fails loudly."""
    from paper_2606_01114_b200 import MMError
    with pytest.raises(MMError) as ei:
        make_ctx(cfg_for((64, 64, 8)), "f64", terms=1, path=2)
    assert ei.value.status == 2
    ctx = make_ctx(cfg_for((64, 64, 8)), "f64", terms=1, path=0)
    assert ctx.path_name in ("generic", "embedded")
    ctx.close()


# nz below the capacity of the warp-per-pencil z kernels (64, 128, 256 layers): the missing layers are read as
# zero and the transform runs at period 2 nzt >= 2 nz - 1, the same linear convolution (reading Q27)
MASKED = [(64, 64, 16), (64, 64, 50), (64, 128, 90), (128, 64, 100), (64, 64, 140), (64, 64, 200), (64, 64, 35)]


@pytest.mark.parametrize("n", MASKED)
def test_fast_fewer_layers_than_the_z_transform(oracle, n):
    cfg = cfg_for(n)
    m32 = w.random_unit_vectors(717, n).astype(np.float32)
    m64 = m32.astype(np.float64)
    P = make_problem(oracle, cfg, terms=1)
    ref = oracle.demag_fft(P.Nhat, cfg.Ms, m64)
    for dt in ("f32", "f64"):
        ctx = make_ctx(cfg, dt, terms=1)
        # an odd nz in fp32 gives pencils that are no multiple of 16 bytes: embedded in nz + 1 layers
        assert ctx.path_name == ("embedded" if (dt == "f32" and n[2] % 2) else "fast"), (n, dt)
        md = to_dev(m64.astype(np.float32 if dt == "f32" else np.float64))
        got = ctx.demag_field(md).cpu().numpy()
        l2, mx = w.field_errors(got, ref)
        assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (n, dt, l2, mx)
        assert np.array_equal(got, ctx.demag_field(md).cpu().numpy())
        ctx.close()


_LDG_WORKER = r"""
import sys
import numpy as np
import torch
sys.path.insert(0, sys.argv[1]); sys.path.insert(0, sys.argv[1] + "/tests")
import workloads as w
from gpu_util import make_ctx, round_input, to_dev
from test_gpu_fast import cfg_for
out = {}
for spec in sys.argv[3:]:
    nx, ny, nz, dt = spec.split(",")
    n = (int(nx), int(ny), int(nz))
    ctx = make_ctx(cfg_for(n), dt, terms=1, path=2)
    m, _ = round_input(w.random_unit_vectors(717, n), dt)
    out[spec] = ctx.demag_field(to_dev(m)).cpu().numpy()
    names = [ctx.kernel_name(k) for k in range(5)]
    assert not any("tma" in s for s in names), names
    ctx.close()
np.savez(sys.argv[2], **out)
"""


def test_tma_box_kernels_bit_identical_to_ldg_kernels(tmp_path):
    """K1, K2, K4, K5 with their tiles moved by 2D TMA boxes (demag_tma.cu) run the stage arithmetic of the
    LDG / STG kernels (demag_fast2.cu) in the same order: the fields must agree bit for bit.  The LDG / STG
    kernels run in a child process with MM_B200_TMA=0 (the switch is read once per process)."""
    import os
    import subprocess
    import sys
    specs = ["64,128,16,f32", "128,64,32,f64", "100,64,24,f32", "256,100,40,f64", "64,350,16,f64", "400,64,32,f32",
             "512,128,16,f32", "64,64,18,f32"]
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    npz = str(tmp_path / "ldg.npz")
    env = dict(os.environ, MM_B200_TMA="0")
    r = subprocess.run([sys.executable, "-c", _LDG_WORKER, root, npz, *specs], env=env, capture_output=True, text=True)
    assert r.returncode == 0, r.stderr[-2000:]
    ref = np.load(npz)
    n_tma = 0
    for spec in specs:
        nx, ny, nz, dt = spec.split(",")
        n = (int(nx), int(ny), int(nz))
        ctx = make_ctx(cfg_for(n), dt, terms=1, path=2)
        n_tma += sum("tma" in ctx.kernel_name(k) for k in range(5))
        m, _ = round_input(w.random_unit_vectors(717, n), dt)
        got = ctx.demag_field(to_dev(m)).cpu().numpy()
        assert np.array_equal(got, ref[spec]), spec
        ctx.close()
    # 64x64x18 fp32 has rows that are not sector aligned (LDG / STG there); nx = 400 keeps the LDG / STG x passes
    assert n_tma >= 4 * (len(specs) - 2) + 2


@pytest.mark.parametrize("spec", ["128,64,64,f64", "64,128,64,f64", "256,128,32,f32", "1024,64,16,f64", "64,1024,16,f32",
                                  "1024,1024,16,f32"])
def test_persistent_box_kernels_are_race_free_over_many_calls(spec):
    """The persistent TMA kernels prefetch the next tile into a buffer the threads have just read.  Without a
    proxy fence before the barrier the box load was seen to overwrite a row ahead of its read about once in
    1e5 tiles (fp64, several CTAs per SM): 600 calls of a mesh whose CTAs walk several tiles must give one
    result."""
    import torch
    nx, ny, nz, dt = spec.split(",")
    n = (int(nx), int(ny), int(nz))
    ctx = make_ctx(cfg_for(n), dt, terms=1, path=2)
    m, _ = round_input(w.random_unit_vectors(717, n), dt)
    md = to_dev(m)
    ref = ctx.demag_field(md).clone()
    out = torch.empty_like(md)
    bad = 0
    for _ in range(600 if n[0] * n[1] < 1e6 else 150):
        ctx.demag_field(md, out)
        bad += int(not torch.equal(out, ref))
    ctx.close()
    assert bad == 0


@pytest.mark.parametrize("n", [(64, 1024, 18), (1024, 100, 18)])
def test_three_stage_passes_with_a_column_tail(oracle, n):
    """L = 1024 (three-stage strided kernels) with rows whose 3 nz complex columns (y passes) or ny 3 nz / 2 pairs
    (x passes) do not fill the last 64-byte tile: the tail columns must be transformed too (round 1 launched
    floor(Q / B) tiles and left them untouched: NaN / O(1) errors at 64x1024x18)."""
    cfg = cfg_for(n)
    P = make_problem(oracle, cfg, terms=1)
    m64 = w.random_unit_vectors(606, n)
    for dt in ("f32", "f64"):
        m, mr = round_input(m64, dt)
        ref = oracle.demag_fft(P.Nhat, cfg.Ms, mr)
        ctx = make_ctx(cfg, dt, terms=1, path=2)
        l2, mx = w.field_errors(ctx.demag_field(to_dev(m)).cpu().numpy(), ref)
        ctx.close()
        assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (n, dt, l2, mx)


@pytest.mark.parametrize("n", [(100, 350, 18), (350, 64, 30), (400, 128, 42), (512, 100, 54), (256, 400, 70),
                               (128, 512, 98), (1024, 64, 20), (64, 1024, 28), (1024, 1024, 18), (100, 1024, 50)])
def test_fast_path_agrees_with_generic_passes_on_ragged_shapes(n):
    """Mixed sides and layer counts that leave partial tiles in every strided pass and partial pencils in K3:
    the x-first kernels against the generic z-first passes (themselves checked against the oracle), both dtypes."""
    cfg = cfg_for(n)
    for dt in ("f32", "f64"):
        m, _ = round_input(w.random_unit_vectors(707, n), dt)
        md = to_dev(m)
        ctx = make_ctx(cfg, dt, terms=1)
        assert ctx.path_name == "fast"
        got = ctx.demag_field(md).cpu().numpy()
        ctx.close()
        ctx = make_ctx(cfg, dt, terms=1, path=1)
        ref = ctx.demag_field(md).cpu().numpy().astype(np.float64)
        ctx.close()
        l2, mx = w.field_errors(got, ref)
        assert np.isfinite(l2) and l2 <= TOL[dt], (n, dt, l2, mx)

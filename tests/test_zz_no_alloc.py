"""mm_demag_field_static (include/mm_b200.h): the demag convolution with its spectra in the library's
file-scope static device array, for callers that cannot allocate.  Checked against the existing path
(mm_demag_field, spectra in the caller's scratch workspace) on two calls in a row, on every demag path
the entry point serves, within the tolerance of the other GPU tests (gpu_util.TOL) -- and, because both
run the same deterministic kernels, bit for bit.  Collected last (test_zz_*): the suite runs with
pytest -x."""
import numpy as np
import pytest
import torch

import workloads as w
from gpu_util import TOL, make_ctx, round_input, to_dev

pytestmark = pytest.mark.gpu

MM_ERR_WORKSPACE, MM_ERR_NOT_IMPLEMENTED = 4, 6
CAPACITY = 32 << 20


def cfg_for(n, d=(4e-9, 3e-9, 2e-9)):
    base = w.get_config(1)
    return w.Config(**{**base.__dict__, "n": n, "d": d, "name": "t"})


def check_pair(ctx, n, dt, seeds):
    """Two calls in a row of the static entry point, each against the existing path on the same input."""
    H = torch.empty(n + (3,), dtype=torch.float32 if dt == "f32" else torch.float64, device="cuda")
    for seed in seeds:
        m, _ = round_input(w.random_unit_vectors(seed, n), dt)
        md = to_dev(m)
        ref = ctx.demag_field(md).cpu().numpy()
        H.fill_(float("nan"))
        got = ctx.demag_field_static(md, out=H).cpu().numpy()
        assert np.isfinite(got).all()
        l2, mx = w.field_errors(got, ref.astype(np.float64))
        assert l2 <= TOL[dt] and mx <= 10 * TOL[dt], (l2, mx)
        assert np.array_equal(got, ref)          # same kernels, fixed summation order: identical bits


# (mesh, dtype, path request, path that runs); 64^3 fp32 is the largest cube the array holds (19.2 MB of 32 MiB)
CASES = [((64, 64, 64), "f32", 2, "fast"), ((64, 64, 16), "f64", 2, "fast"), ((128, 64, 32), "f32", 3, "mixed"),
         ((25, 14, 6), "f64", 3, "mixed"), ((20, 12, 6), "f32", 1, "generic"), ((16, 16, 2), "f64", 1, "generic"),
         ((100, 25, 1), "f32", 0, "generic")]


@pytest.mark.parametrize("n,dt,path,name", CASES)
def test_static_matches_existing_path_on_two_calls_in_a_row(n, dt, path, name):
    ctx = make_ctx(cfg_for(n), dt, terms=1, path=path)
    assert ctx.path_name == name
    cap, need = ctx.static_scratch_info()
    assert cap == CAPACITY and 0 < need <= cap
    check_pair(ctx, n, dt, seeds=(71, 72))
    ctx.close()


def test_static_array_is_shared_and_holds_stale_contents():
    """A large mesh, then a small one, then the large one again: each call finds the array full of another
    call's spectra and must not depend on them."""
    big = make_ctx(cfg_for((64, 64, 64)), "f32", terms=1)
    small = make_ctx(cfg_for((16, 8, 4)), "f64", terms=1)
    check_pair(big, (64, 64, 64), "f32", seeds=(5,))
    check_pair(small, (16, 8, 4), "f64", seeds=(6, 7))
    check_pair(big, (64, 64, 64), "f32", seeds=(8,))
    big.close()
    small.close()


def test_static_call_leaves_the_scratch_workspace_alone_and_allocates_nothing():
    n, dt = (64, 64, 32), "f32"
    ctx = make_ctx(cfg_for(n), dt, terms=1)
    assert ctx.path_name == "fast"
    m, _ = round_input(w.random_unit_vectors(9, n), dt)
    md = to_dev(m)
    ref = ctx.demag_field(md)
    H = torch.empty_like(md)
    ctx.static_scratch_info()                     # set-up: address looked up, module resident
    ctx.demag_field_static(md, out=H)             # warm-up: kernel attributes set
    ctx._ws[1].fill_(0xA5)                        # the context's scratch workspace
    torch.cuda.synchronize()
    outs = [torch.zeros_like(md), torch.zeros_like(md)]
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for out in outs:                                          # nothing but the two calls in the measured region
        ctx.demag_field_static(md, out=out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0              # no device memory taken from the driver
    assert all(torch.equal(out, ref) for out in outs)
    assert bool((ctx._ws[1] == 0xA5).all())                   # the spectra did not go to the workspace
    ctx.close()


def test_static_rejects_what_does_not_fit():
    from paper_2606_01114_b200.binding import MMError
    ctx = make_ctx(cfg_for((64, 64, 64)), "f64", terms=1)    # 38.4 MB of spectra
    cap, need = ctx.static_scratch_info()
    assert need > cap == CAPACITY
    md = to_dev(round_input(w.random_unit_vectors(3, (64, 64, 64)), "f64")[0])
    H = torch.zeros_like(md)
    with pytest.raises(MMError) as ei:
        ctx.demag_field_static(md, out=H)
    assert ei.value.status == MM_ERR_WORKSPACE and str(need) in str(ei.value)
    assert not H.any()                                        # nothing was launched
    ctx.demag_field(md, out=H)                                # the context is still usable
    assert H.any()
    ctx.close()


def test_static_rejects_contexts_that_need_more_than_the_spectra():
    from paper_2606_01114_b200.binding import MMError
    n = (16, 16, 4)
    ctx = make_ctx(cfg_for(n), "f64", terms=1)
    Ms = torch.full(n, 8e5, dtype=torch.float64, device="cuda")
    ctx.set_material_cells(Ms, None)
    md = to_dev(round_input(w.random_unit_vectors(4, n), "f64")[0])
    with pytest.raises(MMError) as ei:
        ctx.demag_field_static(md)
    assert ei.value.status == MM_ERR_NOT_IMPLEMENTED
    assert ctx.static_scratch_info()[1] == 0
    ctx.close()


def test_static_call_inside_a_cuda_graph_capture():
    """The caller this entry point is for: a capture, where nothing may allocate.  Set-up (address look-up,
    kernel attributes) happens before the capture; the captured call is replayed on new inputs."""
    n, dt = (64, 64, 32), "f32"
    ctx = make_ctx(cfg_for(n), dt, terms=1)
    ctx.static_scratch_info()
    md = to_dev(round_input(w.random_unit_vectors(21, n), dt)[0])
    H = torch.zeros_like(md)
    ctx.demag_field_static(md, out=H)                       # warm-up outside the capture
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        ctx.use_current_stream()
        with torch.cuda.graph(g, stream=side):
            ctx.demag_field_static(md, out=H)
    torch.cuda.synchronize()
    ctx.use_current_stream()
    for seed in (22, 23):                                   # two replays in a row on fresh inputs
        md.copy_(to_dev(round_input(w.random_unit_vectors(seed, n), dt)[0]))
        H.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(H, ctx.demag_field(md))
    ctx.close()

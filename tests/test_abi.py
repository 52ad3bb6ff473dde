"""The C-ABI library loads and exports every symbol include/mm_b200.h declares; host-only
argument validation (no kernel is launched, no GPU needed)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_01114_b200 import build, load_library
    build.build()
    return load_library()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "mm_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mm_[a-z_0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    syms = declared_symbols()
    assert len(syms) >= 20 and "mm_rk_step" in syms and "mm_demag_field" in syms
    for s in syms:
        assert hasattr(lib, s), s


def test_create_validates_arguments(lib):
    h = C.c_void_p()
    assert lib.mm_ctx_create(16, 16, 2, 5e-9, 5e-9, 3e-9, 1, C.byref(h)) == 0
    p, s = C.c_size_t(), C.c_size_t()
    assert lib.mm_ctx_workspace_bytes(h, C.byref(p), C.byref(s)) == 0
    assert p.value > 0 and s.value > 0
    # not initialised: no workspace yet
    assert lib.mm_demag_init(h) == 3
    assert b"workspace" in lib.mm_last_error(h)
    assert lib.mm_set_terms(h, 64) == 1
    assert lib.mm_ctx_destroy(h) == 0
    assert lib.mm_ctx_create(11, 16, 2, 5e-9, 5e-9, 3e-9, 1, C.byref(h)) == 2     # prime factor 11
    assert b"2^a 3^b 5^c 7^d" in lib.mm_last_error(None)
    assert lib.mm_ctx_create(12, 350, 90, 5e-9, 5e-9, 3e-9, 1, C.byref(h)) == 0   # mixed radix sizes are fine
    assert lib.mm_ctx_destroy(h) == 0
    assert lib.mm_ctx_create(2048, 16, 2, 5e-9, 5e-9, 3e-9, 1, C.byref(h)) == 2   # above the plan
    assert lib.mm_ctx_create(16, 16, 2, 0.0, 5e-9, 3e-9, 1, C.byref(h)) == 1
    assert lib.mm_ctx_create(16, 16, 2, 5e-9, 5e-9, 3e-9, 7, C.byref(h)) == 1
    assert lib.mm_ctx_create(16, 16, 2, 5e-9, 5e-9, 3e-9, 0, None) == 1


def test_workspace_sizes_match_design(lib):
    """Config 4 fp32.  Generic passes: table 6*129*1024*1024*4 B, spectra 3*129*(512+1024)*512*8 B.
    Fast path (selected automatically): octant table 6*513*513*130*4 B (kz pitch nz+2: 16-byte rows for bulk
    copies), A1 513*512*384*8 B, A2 513*1024*384*8 B.  Field-sized scratch arrays: H_demag, two stage states,
    RK4 accumulator, two host-call staging buffers, six RKF45 k arrays, M = Ms_i m for per-cell Ms."""
    fields = 13 * 512 * 512 * 128 * 3 * 4
    p, s = C.c_size_t(), C.c_size_t()
    path = C.c_int()
    for want, table, spectra in (
            (1, 6 * 129 * 1024 * 1024 * 4, 3 * 129 * (512 + 1024) * 512 * 8),
            (0, 6 * 513 * 513 * 130 * 4, 513 * 512 * 384 * 8 + 513 * 1024 * 384 * 8),
            (2, 6 * 513 * 513 * 130 * 4, 513 * 512 * 384 * 8 + 513 * 1024 * 384 * 8)):
        h = C.c_void_p()
        assert lib.mm_ctx_create(512, 512, 128, 4e-9, 4e-9, 4e-9, 0, C.byref(h)) == 0
        assert lib.mm_ctx_set_path(h, want) == 0
        lib.mm_ctx_workspace_bytes(h, C.byref(p), C.byref(s))
        assert table <= p.value < table + (1 << 20)
        assert spectra + fields <= s.value < spectra + fields + (1 << 20)
        assert lib.mm_ctx_path(h, C.byref(path)) == 0
        assert path.value == (0 if want == 1 else 1)
        lib.mm_ctx_destroy(h)
    h = C.c_void_p()
    assert lib.mm_ctx_create(16, 16, 2, 5e-9, 5e-9, 3e-9, 0, C.byref(h)) == 0
    assert lib.mm_ctx_set_path(h, 2) == 2             # fast kernels do not cover thin films
    assert lib.mm_ctx_set_path(h, 3) == 0             # the mixed-radix x-first kernels do
    assert lib.mm_ctx_path(h, C.byref(path)) == 0 and path.value == 2
    assert lib.mm_ctx_set_path(h, 4) == 1
    lib.mm_ctx_destroy(h)
    assert lib.mm_ctx_create(100, 25, 1, 5e-9, 5e-9, 3e-9, 1, C.byref(h)) == 0
    assert lib.mm_ctx_set_path(h, 3) == 2             # one-cell axis: generic passes only
    lib.mm_ctx_destroy(h)


def test_kernel_names_follow_the_selected_path(lib):
    lib.mm_ctx_kernel_name.restype = C.c_char_p
    lib.mm_ctx_kernel_name.argtypes = [C.c_void_p, C.c_int]
    h = C.c_void_p()
    assert lib.mm_ctx_create(512, 512, 128, 4e-9, 4e-9, 4e-9, 0, C.byref(h)) == 0
    names = [lib.mm_ctx_kernel_name(h, k).decode() for k in range(8)]
    # the y passes run the TMA box kernels where the driver offers cuTensorMapEncodeTiled (not on a CPU-only box)
    assert names[1] in ("yf2_kernel", "yf2_tma_kernel") and names[3] in ("yi2_kernel", "yi2_tma_kernel")
    assert names[0::2] == ["xf2_kernel", "zp_fast_kernel", "xi2_kernel", ""] and names[5] == "pw_vec_kernel" and names[7] == ""
    lib.mm_ctx_destroy(h)
    assert lib.mm_ctx_create(1024, 64, 256, 4e-9, 4e-9, 4e-9, 1, C.byref(h)) == 0
    names = [lib.mm_ctx_kernel_name(h, k).decode() for k in range(5)]
    assert names[0::2] == ["xf_fast_kernel", "zw_fast_kernel", "xi_fast_kernel"] and names[1].startswith("yf2_")
    lib.mm_ctx_destroy(h)
    assert lib.mm_ctx_create(16, 16, 2, 5e-9, 5e-9, 3e-9, 1, C.byref(h)) == 0
    assert lib.mm_ctx_kernel_name(h, 2) == b"xp_kernel" and lib.mm_ctx_kernel_name(h, 5) == b"pw_vec_kernel"
    lib.mm_ctx_destroy(h)


def test_oversized_axis_is_rejected_before_planning(lib):
    """A length whose radix plan would overflow the stage array is refused by the range check, not by
    writing past the plan (n = 2^27 needs nine radix-8 stages)."""
    h = C.c_void_p()
    assert lib.mm_ctx_create(1 << 27, 16, 2, 5e-9, 5e-9, 3e-9, 1, C.byref(h)) == 2
    assert lib.mm_ctx_create(16, 16, 1 << 27, 5e-9, 5e-9, 3e-9, 1, C.byref(h)) == 2

"""Pins for the oracle's demag field (O2-O5): brute-force agreement of three independent
evaluations (direct sum / literal DFT / own FFT), the survey's exact film values, the
thin-film limit, the trace rule and single-source responses.  CPU only."""
import os

import numpy as np
import pytest

import workloads as w

GOLD = os.path.join(os.path.dirname(__file__), "golden", "demag_film_survey_values.txt")


@pytest.mark.parametrize("n,d", [((16, 16, 2), (5e-9, 5e-9, 3e-9)), ((8, 4, 1), (3e-9, 4e-9, 5e-9)),
                                 ((4, 1, 8), (2e-9, 2e-9, 1e-9)), ((1, 1, 4), (1e-9, 2e-9, 3e-9)),
                                 ((1, 1, 1), (1e-9, 2e-9, 3e-9)),
                                 # not powers of two: O4 keeps the paper's period 2n, O5 pads to the next
                                 # power of two (reading Q27); both must equal the direct sum
                                 ((6, 5, 3), (3e-9, 4e-9, 5e-9)), ((7, 3, 2), (2e-9, 2e-9, 1e-9)),
                                 ((12, 10, 1), (5e-9, 5e-9, 3e-9))])
def test_direct_vs_dft_vs_fft(oracle, n, d):
    Ms = 8.0e5
    m = w.random_unit_vectors(77, n)
    N = oracle.newell_octant(n, d)
    Hd = oracle.demag_direct(N, Ms, m)
    Hdft = oracle.demag_dft(N, Ms, m)
    Nhat, max_imag = oracle.demag_fft_nhat(N, return_max_imag=True)
    Hfft = oracle.demag_fft(Nhat, Ms, m)
    assert max_imag < 1e-13                       # Nhat is analytically real
    assert w.field_errors(Hdft, Hd)[1] < 2e-14
    assert w.field_errors(Hfft, Hd)[1] < 2e-14
    assert np.max(np.abs(Hd)) > 0.05 * Ms


def test_single_source_is_minus_Ms_N_m(oracle):
    """One magnetised cell: H(i) = -Ms N(i-j) m_j, the tensor read off directly (sign O2)."""
    n, d, Ms = (8, 8, 4), (5e-9, 5e-9, 3e-9), 1.0e6
    N = oracle.newell_octant(n, d)
    Nhat = oracle.demag_fft_nhat(N)
    src = (5, 2, 1)
    for c in range(3):
        m = np.zeros(n + (3,))
        m[src + (c,)] = 1.0
        for H in (oracle.demag_direct(N, Ms, m), oracle.demag_fft(Nhat, Ms, m)):
            for tgt in [(5, 2, 1), (0, 0, 0), (7, 7, 3), (2, 6, 0), (6, 1, 3)]:
                off = tuple(t - s for t, s in zip(tgt, src))
                Np = oracle.newell_point(d, *off)   # literal, handles signed offsets
                full = np.array([[Np[0], Np[3], Np[4]], [Np[3], Np[1], Np[5]], [Np[4], Np[5], Np[2]]])
                assert np.allclose(H[tgt], -Ms * full[:, c], rtol=1e-12, atol=1e-9 * Ms * 1e-6)
    # self term is positive-definite: H antiparallel to m in the source cell
    assert oracle.demag_direct(N, Ms, m)[src + (2,)] < 0


def _film_rows():
    rows = []
    for line in open(GOLD):
        line = line.split("#")[0].split()
        if line:
            rows.append((int(line[0]), "xyz".index(line[1]), "xyz".index(line[2]), float(line[3])))
    return rows


@pytest.mark.parametrize("W,cm,ch,val", _film_rows())
def test_uniform_film_centre_value(oracle, W, cm, ch, val):
    n, d, Ms = (W, W, 1), (2e-9, 2e-9, 2e-9), 8.0e5
    N = oracle.newell_octant(n, d)
    m = np.zeros(n + (3,))
    m[..., cm] = 1.0
    cell = np.array([(W // 2 * W + W // 2) * 1], dtype=np.int64)
    H = oracle.demag_direct_sampled(N, Ms, m, cell)[0]
    assert H[ch] / Ms == pytest.approx(val, rel=1e-12)
    Hf = oracle.demag_fft(oracle.demag_fft_nhat(N), Ms, m)[W // 2, W // 2, 0]
    assert Hf[ch] / Ms == pytest.approx(val, rel=1e-11)


def test_thin_film_limit(oracle):
    """H -> -Ms m_z deep inside a wide thin out-of-plane film (BASELINE north_star)."""
    Ms = 8.0e5
    prev = 0.0
    for W in (32, 128, 256):
        n, d = (W, W, 1), (4e-9, 4e-9, 1e-9)
        m = np.zeros(n + (3,))
        m[..., 2] = 1.0
        H = oracle.demag_fft(oracle.demag_fft_nhat(oracle.newell_octant(n, d)), Ms, m)
        hz = H[W // 2, W // 2, 0, 2] / Ms
        assert hz < prev or prev == 0.0
        assert -1.0 < hz < -0.9
        assert abs(H[W // 2, W // 2, 0, 0]) < 1e-9 * Ms
        last = hz
    assert last < -0.995


def test_trace_rule_and_nhat_zero(oracle):
    """sum_d -H_d(i).e_d / Ms = 1 at every cell for the three uniform states; Nhat(0) has
    trace 1 (sum of the real-space diagonal)."""
    n, d, Ms = (16, 16, 2), (5e-9, 5e-9, 3e-9), 8.0e5
    N = oracle.newell_octant(n, d)
    Nhat = oracle.demag_fft_nhat(N)
    tot = np.zeros(n)
    for c in range(3):
        m = np.zeros(n + (3,))
        m[..., c] = 1.0
        tot += -oracle.demag_fft(Nhat, Ms, m)[..., c] / Ms
    assert abs(Nhat[0, 0, 0, 0] + Nhat[1, 0, 0, 0] + Nhat[2, 0, 0, 0] - 1.0) < 1e-13
    # survey-computed Nhat(0) for this mesh: diag(0.0261, 0.0261, 0.9478) (SURVEY 8(a) note)
    assert Nhat[0, 0, 0, 0] == pytest.approx(0.0261, abs=5e-5)
    assert Nhat[2, 0, 0, 0] == pytest.approx(0.9478, abs=5e-5)
    # self term has trace 1, every off-site term is traceless => exactly 1 at every cell
    assert np.allclose(tot, 1.0, rtol=0, atol=1e-13)


def test_sampled_equals_full_direct(oracle):
    n, d, Ms = (8, 8, 4), (2e-9, 2e-9, 2e-9), 1e6
    N = oracle.newell_octant(n, d)
    m = w.random_unit_vectors(5, n)
    cells = w.sample_cells(9, n, 20)
    Hs = oracle.demag_direct_sampled(N, Ms, m, cells)
    Hd = oracle.demag_direct(N, Ms, m).reshape(-1, 3)
    assert np.array_equal(Hs, Hd[cells])


def test_fft_period(oracle):
    # powers of two keep the paper's 2n; other sizes pad to the next power of two above 2n
    assert [oracle.fft_period(n) for n in (1, 2, 8, 3, 5, 100, 350, 90)] == [1, 4, 16, 8, 16, 256, 1024, 256]


def test_fft_path_on_a_mesh_shaped_like_the_papers_sp4_grid(oracle):
    # n = (100, 25, 1), 5 x 5 x 3 nm cells; sampled direct sum vs the FFT path
    n, d, Ms = (100, 25, 1), (5e-9, 5e-9, 3e-9), 8.0e5
    m = w.random_unit_vectors(5, n)
    N = oracle.newell_octant(n, d)
    H = oracle.demag_fft(oracle.demag_fft_nhat(N), Ms, m)
    cells = np.array([0, 24, 99 * 25, 99 * 25 + 24, 50 * 25 + 12, 1234, 777])
    Hs = oracle.demag_direct_sampled(N, Ms, m, cells)
    assert np.max(np.abs(H.reshape(-1, 3)[cells] - Hs)) < 1e-13 * Ms

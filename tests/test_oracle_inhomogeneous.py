"""Pins for per-cell Ms and A (O14; eq. 2 as div(A grad M); reading Q31).  CPU only."""
import numpy as np
import pytest

import workloads as w

MU0 = 4e-7 * np.pi


def test_uniform_arrays_equal_the_homogeneous_oracle(oracle):
    n, d = (8, 6, 4), (3e-9, 4e-9, 5e-9)
    m = w.random_unit_vectors(21, n)
    kw = dict(n=n, d=d, Ms=8e5, Aex=1.3e-11, Ku=4e5, axis=(0.0, 0.6, 0.8), alpha=0.1, Hext=(1e4, 2e4, 3e4),
              terms=1 | 2 | 4 | 8 | 16 | 32, D=2e-3, stt_p=(0, 0, 1), stt_damp=1e3, stt_field=2e2)
    P0 = oracle.Problem(**kw).prepare()
    P1 = oracle.Problem(Ms_cells=np.full(n, 8e5), A_cells=np.full(n, 1.3e-11), Nhat=P0.Nhat, **kw)
    H0, H1 = P0.heff(m), P1.heff(m)
    assert np.max(np.abs(H1 - H0)) <= 1e-12 * np.max(np.abs(H0))
    assert np.max(np.abs(P1.llg_rhs(m) - P0.llg_rhs(m))) <= 1e-12 * np.max(np.abs(P0.llg_rhs(m)))


def test_exchange_across_an_interface_uses_the_harmonic_mean(oracle):
    """Two-cell chain: H_1 = 2/(mu0 Ms_1) A_12 (m_2 - m_1)/D^2 with A_12 = 2 A_1 A_2/(A_1 + A_2); written out."""
    n, d = (2, 1, 1), (2e-9, 2e-9, 2e-9)
    Ms = np.array([8e5, 4e5]).reshape(n)
    A = np.array([1.0e-11, 3.0e-11]).reshape(n)
    m = np.zeros(n + (3,))
    m[0, 0, 0] = [1, 0, 0]
    m[1, 0, 0] = [0, 1, 0]
    H = oracle.Problem(n=n, d=d, Ms=8e5, Aex=1e-11, terms=2, Ms_cells=Ms, A_cells=A).heff(m)
    A12 = 2 * 1.0e-11 * 3.0e-11 / 4.0e-11
    assert np.allclose(H[0, 0, 0], 2 / (MU0 * 8e5) * A12 * np.array([-1, 1, 0]) / 4e-18, rtol=1e-13)
    assert np.allclose(H[1, 0, 0], 2 / (MU0 * 4e5) * A12 * np.array([1, -1, 0]) / 4e-18, rtol=1e-13)


def test_exchange_forces_cancel_pairwise(oracle):
    """sum_i Ms_i H_ex(i) = (2/mu0) sum_i sum_j A_ij (m_j - m_i)/D^2 = 0 for any m when A_ij = A_ji:
    fails for an asymmetric mean, a wrong Ms_i prefactor or a boundary term."""
    n, d = (6, 5, 4), (2e-9, 3e-9, 4e-9)
    rng = np.random.default_rng(5)
    Ms = rng.uniform(2e5, 1e6, n)
    A = rng.uniform(0.5e-11, 2e-11, n)
    A[2, 1, :] = 0.0                                   # a decoupled row
    m = w.random_unit_vectors(31, n)
    H = oracle.Problem(n=n, d=d, Ms=8e5, Aex=1e-11, terms=2, Ms_cells=Ms, A_cells=A).heff(m)
    tot = np.sum(Ms[..., None] * H, axis=(0, 1, 2))
    assert np.max(np.abs(tot)) <= 1e-12 * np.sum(np.abs(Ms[..., None] * H))
    assert np.all(H[2, 1, :] == 0.0)                   # A_i = 0: no exchange field


def test_vacuum_cells_do_not_source_the_demag_field_and_do_not_move(oracle):
    """A magnet occupying x < 4 of an 8-cell-long mesh (Ms = 0 elsewhere): the demag field inside equals the
    direct sum O3 over the 4-cell-long magnet alone; vacuum cells have dm/dt = 0 and stay zero under RK4."""
    n, ns, d, Ms0 = (8, 4, 2), (4, 4, 2), (3e-9, 3e-9, 2e-9), 8e5
    m = w.random_unit_vectors(41, n)
    Ms = np.zeros(n)
    Ms[:4] = Ms0
    m[4:] = 0.0
    P = oracle.Problem(n=n, d=d, Ms=Ms0, Aex=1.3e-11, alpha=0.5, terms=1 | 2, Ms_cells=Ms).prepare()
    Hd = oracle.Problem(n=n, d=d, Ms=Ms0, terms=1, Ms_cells=Ms, Nhat=P.Nhat).heff(m)
    ref = oracle.demag_direct(oracle.newell_octant(ns, d), Ms0, m[:4])
    assert np.max(np.abs(Hd[:4] - ref)) <= 1e-13 * Ms0
    k = P.llg_rhs(m)
    assert np.all(k[4:] == 0.0) and np.max(np.abs(k[:4])) > 0
    m1 = P.rk4_step(m, 1e-13)
    assert np.all(m1[4:] == 0.0) and np.max(np.abs(np.linalg.norm(m1[:4], axis=-1) - 1)) < 1e-14
    # the surface cell x = 3 sees no exchange partner at x = 4 (A_ij with a vacuum... A is uniform here, but
    # the neighbour's m is zero): with A_cells zero in vacuum the interface term drops as at a mesh boundary
    A = np.where(Ms > 0, 1.3e-11, 0.0)
    Hx = oracle.Problem(n=n, d=d, Ms=Ms0, Aex=1.3e-11, terms=2, Ms_cells=Ms, A_cells=A).heff(m)
    ref_x = oracle.exchange(d, Ms0, 1.3e-11, m[:4])
    assert np.max(np.abs(Hx[:4] - ref_x)) <= 1e-13 * np.max(np.abs(ref_x))
    # the same holds with UNIFORM A (A_cells = None) and arbitrary non-zero vectors stored in the vacuum
    # cells: a neighbour with Ms_j = 0 is no exchange partner (reading Q31), so the magnet's exchange
    # field is that of the 4-cell-long mesh and does not depend on what the vacuum cells hold
    mv = m.copy()
    mv[4:] = w.random_unit_vectors(43, n)[4:]
    Hu = oracle.Problem(n=n, d=d, Ms=Ms0, Aex=1.3e-11, terms=2, Ms_cells=Ms).heff(mv)
    assert np.max(np.abs(Hu[:4] - ref_x)) <= 1e-13 * np.max(np.abs(ref_x))
    assert np.all(Hu[4:] == 0.0)


def test_demag_is_linear_in_Ms_cells_and_dmi_skips_vacuum_neighbours(oracle):
    n, d = (6, 4, 2), (2e-9, 2e-9, 2e-9)
    m = w.random_unit_vectors(51, n)
    rng = np.random.default_rng(6)
    Ms = rng.uniform(2e5, 1e6, n)
    P = oracle.Problem(n=n, d=d, Ms=8e5, terms=1, Ms_cells=Ms).prepare()
    P2 = oracle.Problem(n=n, d=d, Ms=8e5, terms=1, Ms_cells=2.5 * Ms, Nhat=P.Nhat)
    assert np.allclose(P2.heff(m), 2.5 * P.heff(m), rtol=1e-13, atol=1e-9)
    # DMI: with Ms = 0 beyond x = 2 the cell x = 2 sees the half slope of a surface cell
    Ms2 = np.full(n, 8e5)
    Ms2[3:] = 0.0
    lin = np.zeros(n + (3,))
    lin[..., 2] = (1e7 * 2e-9 * np.arange(n[0])).reshape(-1, 1, 1)
    H = oracle.Problem(n=n, d=d, Ms=8e5, terms=16, D=3e-3, Ms_cells=Ms2).heff(lin)
    pref = 2 * 3e-3 / (MU0 * 8e5)
    assert np.allclose(H[1, :, :, 0], pref * 1e7, rtol=1e-12) and np.allclose(H[2, :, :, 0], 0.5 * pref * 1e7, rtol=1e-12)
    assert np.all(H[3:] == 0.0)

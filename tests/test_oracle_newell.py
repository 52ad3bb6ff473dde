"""Pins for the oracle's Newell tensor (O1): closed forms, the survey's independent mpmath
values, the far-field dipole, symmetry/trace invariants and a Gauss-Legendre quadrature of
the defining surface-charge integral (an evaluation that shares nothing with the f/g closed
forms).  CPU only."""
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden", "newell_survey_values.txt")
COMP = {"xx": 0, "yy": 1, "zz": 2, "xy": 3, "xz": 4, "yz": 5}


def _rows():
    rows = []
    for line in open(GOLD):
        line = line.split("#")[0].split()
        if line:
            rows.append((tuple(map(float, line[:3])), tuple(map(int, line[3:6])), line[6],
                         float(line[7])))
    return rows


@pytest.mark.parametrize("d,ijk,comp,val", _rows())
def test_survey_values(oracle, d, ijk, comp, val):
    got = oracle.newell_point(d, *ijk)[COMP[comp]]
    assert got == pytest.approx(val, rel=2e-14, abs=1e-25)


def test_cube_self_term_is_one_third(oracle):
    N = oracle.newell_point((2e-9, 2e-9, 2e-9), 0, 0, 0)
    assert np.allclose(N[:3], 1.0 / 3.0, rtol=0, atol=2e-16)
    assert np.all(N[3:] == 0.0)


@pytest.mark.parametrize("d", [(1, 1, 2), (1, 2, 3), (5e-9, 5e-9, 3e-9), (4, 4, 0.7), (0.3, 7, 2)])
def test_self_trace_is_one(oracle, d):
    N = oracle.newell_point(d, 0, 0, 0)
    assert abs(N[:3].sum() - 1.0) < 4e-16
    if d[0] == d[1]:
        assert N[0] == pytest.approx(N[1], rel=1e-15)


@pytest.mark.parametrize("ijk", [(1, 0, 0), (0, 2, 0), (1, 1, 1), (3, 2, 1), (7, 0, 5), (20, 10, 5)])
@pytest.mark.parametrize("d", [(1, 1, 1), (5, 5, 3), (1, 2, 3)])
def test_offsite_traceless(oracle, ijk, d):
    N = oracle.newell_point(d, *ijk)
    assert abs(N[:3].sum()) < 1e-16 * max(1.0, np.abs(N).max() / 1e-3)


def test_axis_permutation_symmetry(oracle):
    """Permuting the axes of cell and offset permutes the tensor components."""
    a = oracle.newell_point((1, 2, 3), 2, 3, 1)          # xx yy zz xy xz yz
    b = oracle.newell_point((2, 3, 1), 3, 1, 2)          # axes rotated x<-y<-z<-x
    # new x = old y, new y = old z, new z = old x
    assert b[0] == pytest.approx(a[1], rel=1e-13)        # xx' = yy
    assert b[1] == pytest.approx(a[2], rel=1e-13)        # yy' = zz
    assert b[2] == pytest.approx(a[0], rel=1e-13)        # zz' = xx
    assert b[3] == pytest.approx(a[5], rel=1e-13)        # x'y' = yz
    assert b[4] == pytest.approx(a[3], rel=1e-13)        # x'z' = yx
    assert b[5] == pytest.approx(a[4], rel=1e-13)        # y'z' = zx


def test_far_field_is_point_dipole(oracle):
    """N -> -(V/4pi)(3 r_i r_j / r^5 - delta_ij / r^3); cubic cells: error ~ 0.04 R^-7."""
    d = (1.0, 1.0, 1.0)
    for ijk in [(20, 10, 5), (40, 0, 0), (30, 30, 30), (64, 3, 17)]:
        r = np.array(ijk, dtype=float)
        R = np.linalg.norm(r)
        dip = -(1.0 / (4 * np.pi)) * (3 * np.outer(r, r) / R**5 - np.eye(3) / R**3)
        N = oracle.newell_point(d, *ijk)
        full = np.array([[N[0], N[3], N[4]], [N[3], N[1], N[5]], [N[4], N[5], N[2]]])
        assert np.max(np.abs(full - dip)) < 0.2 * R**-7


def test_far_field_noncubic(oracle):
    d = (5.0, 5.0, 3.0)
    V = 75.0
    ijk = (100, 40, 60)
    r = np.array(ijk) * np.array(d)
    R = np.linalg.norm(r)
    dip = -(V / (4 * np.pi)) * (3 * np.outer(r, r) / R**5 - np.eye(3) / R**3)
    N = oracle.newell_point(d, *ijk)
    full = np.array([[N[0], N[3], N[4]], [N[3], N[1], N[5]], [N[4], N[5], N[2]]])
    assert np.max(np.abs(full - dip)) < 1e-3 * np.max(np.abs(dip))


def _gl_tensor_element(d, off, a, b, npts=14):
    """N_ab between a source cell at the origin and a target cell at offset `off` (cells),
    by Gauss-Legendre quadrature of   (1/(4 pi V)) oint_target dS n_a oint_source dS' n'_b / |r-r'|
    (the magnetostatic surface-charge definition; H = -N M averaged over the target cell)."""
    d = np.asarray(d, float)
    X = np.asarray(off, float) * d
    V = d.prod()
    x, w = np.polynomial.legendre.leggauss(npts)
    ta = [q for q in range(3) if q != a]   # in-plane axes of the target face (normal a)
    sb = [q for q in range(3) if q != b]   # in-plane axes of the source face (normal b)
    g = np.meshgrid(x, x, x, x, indexing="ij")
    W = np.einsum("i,j,k,l->ijkl", w, w, w, w)
    jac = (d[ta[0]] / 2) * (d[ta[1]] / 2) * (d[sb[0]] / 2) * (d[sb[1]] / 2)
    total = 0.0
    for s in (+1, -1):
        for sp in (+1, -1):
            rt = [None] * 3
            rs = [None] * 3
            rt[a] = X[a] + s * d[a] / 2
            rt[ta[0]] = X[ta[0]] + g[0] * d[ta[0]] / 2
            rt[ta[1]] = X[ta[1]] + g[1] * d[ta[1]] / 2
            rs[b] = sp * d[b] / 2
            rs[sb[0]] = g[2] * d[sb[0]] / 2
            rs[sb[1]] = g[3] * d[sb[1]] / 2
            dist = np.sqrt(sum((rt[q] - rs[q]) ** 2 for q in range(3)))
            total += s * sp * np.sum(W / dist) * jac
    return total / (4 * np.pi * V)


@pytest.mark.parametrize("d,off", [((1, 1, 1), (2, 0, 0)), ((1, 1, 1), (3, 2, 1)),
                                   ((5, 5, 3), (2, 1, 2)), ((1, 2, 3), (2, 2, 1)),
                                   ((3.90625, 3.90625, 3), (4, 3, 0))])
def test_against_quadrature_of_definition(oracle, d, off):
    N = oracle.newell_point(d, *off)
    pairs = {0: (0, 0), 1: (1, 1), 2: (2, 2), 3: (0, 1), 4: (0, 2), 5: (1, 2)}
    for comp, (a, b) in pairs.items():
        q = _gl_tensor_element(d, off, a, b)
        assert N[comp] == pytest.approx(q, rel=1e-8, abs=1e-11), (comp, N[comp], q)


def test_octant_table_matches_literal_definition(oracle):
    """The lattice-regrouped table equals the literal 27-point evaluation, entry by entry."""
    n, d = (6, 5, 4), (5e-9, 4e-9, 3e-9)
    N = oracle.newell_octant(n, d)
    for ijk in [(0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), (5, 4, 3), (2, 3, 1), (5, 0, 2), (0, 4, 3)]:
        lit = oracle.newell_point(d, *ijk)
        tab = N[(slice(None),) + ijk]
        assert np.allclose(tab, lit, rtol=1e-15, atol=1e-30)


def test_structural_zeros(oracle):
    N = oracle.newell_octant((4, 4, 4), (1, 1, 1))
    assert np.all(N[3, 0, :, :] == 0) and np.all(N[3, :, 0, :] == 0)
    assert np.all(N[4, 0, :, :] == 0) and np.all(N[4, :, :, 0] == 0)
    assert np.all(N[5, :, 0, :] == 0) and np.all(N[5, :, :, 0] == 0)
    assert np.all(N[3, 1:, 1:, :] != 0)

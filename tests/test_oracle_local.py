"""Pins for the oracle's local terms, LLG right-hand side and RK4 (O6-O9): closed forms and
invariants from SURVEY.md 8(c).  CPU only."""
import numpy as np
import pytest

import workloads as w

MU0 = 4e-7 * np.pi


def test_exchange_zero_for_uniform(oracle):
    m = np.zeros((6, 5, 4, 3))
    m[...] = np.array([0.6, 0.0, 0.8])
    H = oracle.exchange((1e-9, 2e-9, 3e-9), 8e5, 1.3e-11, m)
    assert np.all(H == 0.0)


@pytest.mark.parametrize("axis,q", [(0, 1), (0, 3), (1, 2), (2, 1)])
def test_exchange_neumann_eigenvector(oracle, axis, q):
    """m_x(j) = cos(pi q (j+1/2)/n)  =>  H_x = -(2A/mu0 Ms)(4/D^2) sin^2(pi q/2n) m_x exactly."""
    n = (8, 6, 4)
    d = (1e-9, 2e-9, 3e-9)
    Ms, A = 8e5, 1.3e-11
    j = np.arange(n[axis])
    prof = np.cos(np.pi * q * (j + 0.5) / n[axis])
    shape = [1, 1, 1]
    shape[axis] = n[axis]
    m = np.zeros(n + (3,))
    m[..., 0] = prof.reshape(shape)
    m[..., 1] = 0.25                                  # uniform component: no contribution
    H = oracle.exchange(d, Ms, A, m)
    lam = -(2 * A / (MU0 * Ms)) * (4 / d[axis] ** 2) * np.sin(np.pi * q / (2 * n[axis])) ** 2
    assert np.allclose(H[..., 0], lam * m[..., 0], rtol=1e-12, atol=1e-9 * abs(lam))
    assert np.allclose(H[..., 1], 0.0, atol=1e-9 * abs(lam))
    assert np.all(H[..., 2] == 0.0)


def test_exchange_single_axis_contributes_nothing(oracle):
    m = w.random_unit_vectors(3, (1, 1, 1))
    assert np.all(oracle.exchange((1e-9,) * 3, 8e5, 1e-11, m) == 0.0)
    m = w.random_unit_vectors(3, (4, 1, 1))
    H = oracle.exchange((1e-9, 5e-9, 7e-9), 8e5, 1e-11, m)
    # hand stencil, first cell: neighbour on the left replaced by itself
    pref = 2 * 1e-11 / (MU0 * 8e5) / 1e-18
    assert np.allclose(H[0, 0, 0], pref * (m[1, 0, 0] - m[0, 0, 0]), rtol=1e-13)
    assert np.allclose(H[2, 0, 0], pref * (m[3, 0, 0] - 2 * m[2, 0, 0] + m[1, 0, 0]), rtol=1e-12)


def test_anisotropy_closed_forms(oracle):
    Ms, Ku = 1e6, 5e5
    u = np.array([0.0, 0.0, 1.0])
    m = np.zeros((2, 1, 1, 3))
    m[0, 0, 0] = u
    m[1, 0, 0] = [1.0, 0.0, 0.0]
    H = oracle.anisotropy(Ms, Ku, u, m)
    assert np.allclose(H[0, 0, 0], 2 * Ku / (MU0 * Ms) * u, rtol=1e-15)
    assert np.all(H[1, 0, 0] == 0.0)
    u2 = np.array([1.0, 2.0, 2.0]) / 3.0
    mm = w.random_unit_vectors(1, (3, 3, 3))
    H = oracle.anisotropy(Ms, Ku, u2, mm)
    assert np.allclose(H, 2 * Ku / (MU0 * Ms) * (mm @ u2)[..., None] * u2, rtol=1e-13)


def test_llg_hand_example_and_invariants(oracle):
    alpha, gamma, h = 0.3, 2.211e5, 1.0e5
    m = np.array([[[[1.0, 0.0, 0.0]]]])
    H = np.array([[[[0.0, h, 0.0]]]])
    # m x H = h z ;  m x (m x H) = x x (h z) = -h y
    want = -gamma / (1 + alpha**2) * np.array([0.0, -alpha * h, h])
    assert np.allclose(oracle.llg_torque(alpha, gamma, m, H)[0, 0, 0], want, rtol=1e-15)
    mm = w.random_unit_vectors(11, (4, 4, 4))
    HH = 1e6 * w.normal_field(12, 4 * 4 * 4 * 3).reshape(4, 4, 4, 3)
    t = oracle.llg_torque(alpha, gamma, mm, HH)
    assert np.max(np.abs(np.sum(mm * t, axis=-1))) < 1e-15 * np.max(np.abs(t))   # m . dm/dt = 0
    # H || m -> 0 (round-off of gamma*|H| only)
    assert np.max(np.abs(oracle.llg_torque(alpha, gamma, mm, 3e5 * mm))) < 1e-15 * gamma * 3e5


def _macrospin(oracle, dt, steps, alpha=0.1, Hz=1e6):
    P = oracle.Problem(n=(2, 1, 1), d=(1e-9,) * 3, Ms=8e5, alpha=alpha, Hext=(0, 0, Hz),
                       terms=oracle.TERM_ZEEMAN)
    m0 = np.array([np.sin(1.0), 0.0, np.cos(1.0)])
    m = np.tile(m0, (2, 1, 1, 1))
    for _ in range(steps):
        m = P.rk4_step(m, dt)
    T = dt * steps
    g = 2.211e5
    mz = np.tanh(alpha * g * Hz * T / (1 + alpha**2) + np.arctanh(m0[2]))
    phi = g * Hz * T / (1 + alpha**2)
    s = np.sqrt(1 - mz * mz)
    exact = np.array([s * np.cos(phi), s * np.sin(phi), mz])
    return np.max(np.abs(m[0, 0, 0] - exact)), m


def test_rk4_macrospin_closed_form_and_order(oracle):
    """Uniform m in a constant field: m_z = tanh(a g H t/(1+a^2) + atanh m_z0), azimuth
    g H t/(1+a^2); the global error of RK4 falls 16x when dt halves."""
    e4, _ = _macrospin(oracle, 4e-13, 50)
    e2, _ = _macrospin(oracle, 2e-13, 100)
    e1, m = _macrospin(oracle, 1e-13, 200)
    assert e1 < 1e-8 and e2 < 2e-7
    assert 12 < e4 / e2 < 20 and 12 < e2 / e1 < 20
    assert np.allclose(np.linalg.norm(m, axis=-1), 1.0, atol=1e-15)


def test_heff_is_sum_of_terms(oracle):
    c = w.get_config(1)
    m = c.initial_m()
    P = oracle.Problem(n=c.n, d=c.d, Ms=c.Ms, Aex=c.Aex, Ku=2e5, axis=(0, 0.6, 0.8), alpha=c.alpha,
                       Hext=(1e4, -2e4, 3e4), terms=15).prepare()
    H = P.heff(m)
    parts = (oracle.demag_fft(P.Nhat, c.Ms, m) + oracle.exchange(c.d, c.Ms, c.Aex, m)
             + oracle.anisotropy(c.Ms, 2e5, (0, 0.6, 0.8), m) + np.array([1e4, -2e4, 3e4]))
    assert np.allclose(H, parts, rtol=1e-14, atol=1e-6)
    assert np.allclose(P.llg_rhs(m), oracle.llg_torque(c.alpha, 2.211e5, m, H), rtol=1e-14)


def test_rk4_conserves_norm_full_problem(oracle):
    c = w.get_config(1)
    P = oracle.Problem(n=c.n, d=c.d, Ms=c.Ms, Aex=c.Aex, alpha=c.alpha, terms=c.terms).prepare()
    m = c.initial_m()
    m1 = P.rk4_step(m, c.dt)
    assert np.allclose(np.linalg.norm(m1, axis=-1), 1.0, atol=2e-16)
    assert 0 < np.max(np.abs(m1 - m)) < 0.5


# ---------------------------------------------------------------- O10: RKF45

def _precession_problem(oracle, alpha, Hz=1e6):
    return oracle.Problem(n=(2, 1, 1), d=(1e-9,) * 3, Ms=8e5, alpha=alpha, Hext=(0, 0, Hz),
                          terms=oracle.TERM_ZEEMAN)


def test_rkf45_linear_precession_matches_stability_polynomials(oracle):
    """alpha = 0, uniform m in H = H z: m_x + i m_y obeys y' = i g H y, a linear test equation.
    One RKF45 step multiplies y by the pair's stability polynomials (Hairer-Norsett-Wanner, Fehlberg
    4(5)): R5(z) = 1 + z + z^2/2 + z^3/6 + z^4/24 + z^5/120 + z^6/2080 and
    R4(z) = 1 + ... + z^4/24 + z^5/104, z = i g H dt.  So the accepted state has azimuth arg R5(z)
    (renormalisation only rescales), m_z unchanged, and the error estimate is
    s max(|Re|, |Im|) of (R5 - R4)(z) = s max(|z|^6/2080, |z|^5 (1/104 - 1/120))."""
    P = _precession_problem(oracle, 0.0)
    th = 0.9
    s, mz = np.sin(th), np.cos(th)
    m0 = np.tile(np.array([s, 0.0, mz]), (2, 1, 1, 1))
    for dt in (2e-12, 1e-12, 3e-13):
        x = 2.211e5 * 1e6 * dt
        z = 1j * x
        R5 = 1 + z + z**2 / 2 + z**3 / 6 + z**4 / 24 + z**5 / 120 + z**6 / 2080
        m1, err, acc, _ = P.rkf45_step(m0, dt, tol=1.0, dt_min=0.0, dt_max=1.0)
        assert acc
        y = s * R5
        want = np.array([y.real, y.imag, mz])
        want /= np.linalg.norm(want)
        assert np.allclose(m1[0, 0, 0], want, rtol=0, atol=3e-16)
        est = s * max(x**6 / 2080, x**5 * (1 / 104 - 1 / 120))
        assert abs(err - est) <= 1e-12 * est + 2e-16, (dt, err, est)


def test_rkf45_macrospin_fifth_order_and_estimate_scaling(oracle):
    """Damped macrospin (closed form as for RK4): with the step held fixed the propagated
    5th-order solution has global error falling 32x when dt halves, and the error estimate of a
    single step (a 4th-order local error) falls 32x as well."""
    P = _precession_problem(oracle, 0.1)
    m0 = np.array([np.sin(1.0), 0.0, np.cos(1.0)])
    g, Hz, alpha = 2.211e5, 1e6, 0.1

    def run(dt, steps):
        m = np.tile(m0, (2, 1, 1, 1))
        for _ in range(steps):
            m, _, acc, dtn = P.rkf45_step(m, dt, tol=1.0, dt_min=dt, dt_max=dt)
            assert acc and dtn == dt
        T = dt * steps
        mz = np.tanh(alpha * g * Hz * T / (1 + alpha**2) + np.arctanh(m0[2]))
        phi = g * Hz * T / (1 + alpha**2)
        sxy = np.sqrt(1 - mz * mz)
        return np.max(np.abs(m[0, 0, 0] - np.array([sxy * np.cos(phi), sxy * np.sin(phi), mz])))

    e4, e2, e1 = run(4e-12, 10), run(2e-12, 20), run(1e-12, 40)
    assert e1 < 5e-6 and e4 < 2e-3
    assert 24 < e4 / e2 < 40 and 24 < e2 / e1 < 40, (e4, e2, e1)
    m = np.tile(m0, (2, 1, 1, 1))
    errs = [P.rkf45_step(m, dt, tol=1.0)[1] for dt in (4e-12, 2e-12, 1e-12)]
    assert 24 < errs[0] / errs[1] < 40 and 24 < errs[1] / errs[2] < 40, errs


def test_rkf45_step_control(oracle):
    """Readings Q23-Q26: accept iff err <= tol; a rejected attempt leaves m untouched; the factor
    0.9 (tol/err)^(1/5) is clamped to [0.2, 5] and dt to [dt_min, dt_max]."""
    c = w.get_config(1)
    P = oracle.Problem(n=c.n, d=c.d, Ms=c.Ms, Aex=c.Aex, alpha=c.alpha, terms=c.terms).prepare()
    m = c.initial_m()
    dt = 2e-13
    m1, err, acc, dtn = P.rkf45_step(m, dt, tol=1.0)
    assert acc and err > 0 and dtn == 5 * dt                        # huge tol: factor clamp 5
    assert np.allclose(np.linalg.norm(m1, axis=-1), 1.0, atol=2e-16)
    m2, err2, acc2, dtn2 = P.rkf45_step(m, dt, tol=err * 1e-9)
    assert not acc2 and err2 == err and np.array_equal(m2, m)      # rejected: m untouched
    assert dtn2 == 0.2 * dt                                         # factor clamp 0.2
    _, _, acc3, dtn3 = P.rkf45_step(m, dt, tol=err)                # err == tol is accepted
    assert acc3 and abs(dtn3 - 0.9 * dt) < 1e-12 * dt
    _, _, acc4, dtn4 = P.rkf45_step(m, dt, tol=err / 2)
    assert not acc4 and abs(dtn4 - 0.9 * 0.5**0.2 * dt) < 1e-12 * dt
    assert P.rkf45_step(m, dt, tol=1.0, dt_max=3 * dt)[3] == 3 * dt
    assert P.rkf45_step(m, dt, tol=err * 1e-9, dt_min=0.5 * dt)[3] == 0.5 * dt
    # against RK4 (a different 4th-order method): same state to the size of the error estimate
    assert np.max(np.abs(m1 - P.rk4_step(m, dt))) < 50 * err


# ------------------------------------------------------------------ O11 DMI (eq. 3)

def _linear(n, axis, comp, slope, d):
    """m_comp = slope * (coordinate along axis); the stencil is linear per component, so the test
    input need not have unit length."""
    m = np.zeros(n + (3,))
    shape = [1, 1, 1]
    shape[axis] = n[axis]
    m[..., comp] = (slope * d[axis] * np.arange(n[axis])).reshape(shape)
    return m


def test_dmi_zero_for_uniform_and_single_cell_axes(oracle):
    m = np.zeros((5, 4, 3, 3))
    m[...] = np.array([0.6, 0.0, 0.8])
    for e in (oracle.DMI_INTERFACIAL, oracle.DMI_BULK):
        assert np.all(oracle.dmi((1e-9, 2e-9, 3e-9), 8e5, 3e-3, e, m) == 0.0)
    mm = w.random_unit_vectors(4, (1, 1, 1))
    assert np.all(oracle.dmi((1e-9,) * 3, 8e5, 3e-3, oracle.DMI_BULK, mm) == 0.0)


def test_dmi_interfacial_is_the_textbook_field(oracle):
    """e_x = e_y-hat, e_y = -e_x-hat:  sum_k e_k x d_k m =
    (d_x m_z, d_y m_z, -d_x m_x - d_y m_y); interior cells see the exact slope, surface cells
    half of it (missing neighbour := the cell itself)."""
    n, d, Ms, D = (6, 5, 2), (2e-9, 3e-9, 1e-9), 8e5, 3e-3
    pref = 2 * D / (MU0 * Ms)
    cases = [((0, 2, 7e7), (0, 1.0)), ((1, 2, -4e7), (1, 1.0)), ((0, 0, 5e7), (2, -1.0)), ((1, 1, 6e7), (2, -1.0)),
             ((0, 1, 5e7), None), ((1, 0, 5e7), None), ((2, 0, 5e7), None), ((2, 2, 5e7), None)]
    for (axis, comp, slope), expect in cases:
        H = oracle.dmi(d, Ms, D, oracle.DMI_INTERFACIAL, _linear(n, axis, comp, slope, d))
        if expect is None:
            assert np.all(H == 0.0), (axis, comp)
            continue
        oc, sign = expect
        inner = [slice(None)] * 3
        inner[axis] = slice(1, -1)
        assert np.allclose(H[tuple(inner) + (oc,)], sign * pref * slope, rtol=1e-12)
        edge = [slice(None)] * 3
        edge[axis] = 0
        assert np.allclose(H[tuple(edge) + (oc,)], 0.5 * sign * pref * slope, rtol=1e-12)
        others = [c for c in range(3) if c != oc]
        assert np.all(H[..., others] == 0.0)


def test_dmi_bulk_is_the_curl(oracle):
    """e_k = unit vector k: sum_k e_k x d_k m = curl m.  On m = (sin(q y), sin(q z), sin(q x)) the
    central difference of sin is cos * sin(q D)/D exactly (interior cells)."""
    n, d, Ms, D = (9, 8, 7), (1e-9, 1.5e-9, 2e-9), 1e6, 2e-3
    q = 2.0e8
    x = (np.arange(n[0]) * d[0]).reshape(-1, 1, 1)
    y = (np.arange(n[1]) * d[1]).reshape(1, -1, 1)
    z = (np.arange(n[2]) * d[2]).reshape(1, 1, -1)
    m = np.zeros(n + (3,))
    m[..., 0] = np.sin(q * y)
    m[..., 1] = np.sin(q * z)
    m[..., 2] = np.sin(q * x)
    H = oracle.dmi(d, Ms, D, oracle.DMI_BULK, m)
    pref = 2 * D / (MU0 * Ms)
    fd = [np.sin(q * h) / h for h in d]
    curl = np.zeros_like(m)
    curl[..., 0] = 0 * x + 0 * y - np.cos(q * z) * fd[2]      # d_y m_z - d_z m_y
    curl[..., 1] = 0 * y + 0 * z - np.cos(q * x) * fd[0]      # d_z m_x - d_x m_z
    curl[..., 2] = 0 * x + 0 * z - np.cos(q * y) * fd[1]      # d_x m_y - d_y m_x
    inner = (slice(1, -1),) * 3
    assert np.allclose(H[inner], pref * curl[inner], rtol=1e-10, atol=1e-12 * pref * q)


def test_dmi_general_vectors_match_numpy_cross(oracle):
    """Arbitrary e_k on a random field: numpy's gradient-free restatement with np.cross and np.roll."""
    n, d, Ms, D = (5, 4, 3), (1e-9, 2e-9, 3e-9), 8e5, 1e-3
    rng = np.random.default_rng(3)
    e = rng.normal(size=(3, 3))
    m = w.random_unit_vectors(9, n)
    H = oracle.dmi(d, Ms, D, e, m)
    acc = np.zeros_like(m)
    for k in range(3):
        hi = np.concatenate([np.take(m, range(1, n[k]), axis=k), np.take(m, [n[k] - 1], axis=k)], axis=k)
        lo = np.concatenate([np.take(m, [0], axis=k), np.take(m, range(0, n[k] - 1), axis=k)], axis=k)
        acc += np.cross(e[k], (hi - lo) / (2 * d[k]))
    assert np.allclose(H, 2 * D / (MU0 * Ms) * acc, rtol=1e-12, atol=1e-3)


# ------------------------------------------------------------------ O12 spin-torque field

def test_stt_field_closed_forms(oracle):
    p = np.array([0.0, 0.0, 1.0])
    m = np.zeros((3, 1, 1, 3))
    m[0, 0, 0] = [1, 0, 0]
    m[1, 0, 0] = [0, 1, 0]
    m[2, 0, 0] = [0, 0, 1]
    H = oracle.stt(p, 2.0e3, 5.0e2, m)
    assert np.allclose(H[0, 0, 0], [0, -2.0e3, 5.0e2])     # x-hat x z-hat = -y-hat
    assert np.allclose(H[1, 0, 0], [2.0e3, 0, 5.0e2])      # y-hat x z-hat = +x-hat
    assert np.allclose(H[2, 0, 0], [0, 0, 5.0e2])          # m || p: only the field-like part
    mm = w.random_unit_vectors(2, (4, 3, 2))
    pp = np.array([1.0, 2.0, 2.0]) / 3.0
    assert np.allclose(oracle.stt(pp, 7.0, -3.0, mm), 7.0 * np.cross(mm, pp) - 3.0 * pp, rtol=1e-13)


def test_heff_adds_dmi_and_stt(oracle):
    n, d = (6, 4, 2), (2e-9, 2e-9, 1e-9)
    m = w.random_unit_vectors(5, n)
    kw = dict(n=n, d=d, Ms=8e5, Aex=1.3e-11, alpha=0.1)
    base = oracle.Problem(terms=2, **kw).heff(m)
    full = oracle.Problem(terms=2 | 16 | 32, D=3e-3, edmi=oracle.DMI_INTERFACIAL, stt_p=(0, 0, 1),
                          stt_damp=1e3, stt_field=2e2, **kw).heff(m)
    want = base + oracle.dmi(d, 8e5, 3e-3, oracle.DMI_INTERFACIAL, m) + oracle.stt((0, 0, 1), 1e3, 2e2, m)
    assert np.allclose(full, want, rtol=1e-13, atol=1e-6)

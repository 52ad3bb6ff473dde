"""Pins for the oracle's Barzilai-Borwein minimiser O13 (reading Q30):
closed forms of the norm-preserving update, the inverse-curvature property of the BB step, the
Stoner-Wohlfarth hard-axis equilibrium, fixed points, and relaxation of an exchange chain.  CPU only."""
import numpy as np
import pytest

import workloads as w

MU0 = 4e-7 * np.pi


def macrospin(oracle, H=(0.0, 0.0, 1.0e5), Ku=0.0, axis=(0, 0, 1), terms=8):
    return oracle.Problem(n=(1, 1, 1), d=(1e-9,) * 3, Ms=8e5, Ku=Ku, axis=axis, Hext=H, terms=terms)


def unit(theta, phi=0.3):
    return np.array([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)]).reshape(1, 1, 1, 3)


@pytest.mark.parametrize("theta0,tau0", [(1.0, 4e-6), (2.5, 1e-5), (0.2, 5e-6)])
def test_first_step_is_a_rotation_towards_H_by_the_cayley_angle(oracle, theta0, tau0):
    """tau g with g = m x (m x H), |g| = H sin(theta): the update rotates m in the (m, H) plane by
    phi with tan(phi/2) = tau H sin(theta)/2, towards H, and keeps |m| = 1 and the azimuth."""
    Hz = 1.0e5
    bb = oracle.BBMinimizer(macrospin(oracle, (0, 0, Hz)), unit(theta0), tau0=tau0, tau_min=0.0, tau_max=1.0)
    tau, dm, conv = bb.step()
    assert tau == tau0 and not conv
    m1 = bb.m.reshape(3)
    assert abs(np.linalg.norm(m1) - 1.0) < 1e-15
    theta1 = np.arccos(m1[2])
    phi = 2.0 * np.arctan(0.5 * tau0 * Hz * np.sin(theta0))
    assert abs((theta0 - theta1) - phi) < 1e-13
    assert abs(np.arctan2(m1[1], m1[0]) - 0.3) < 1e-13
    assert abs(dm - np.max(np.abs(m1 - unit(theta0).reshape(3)))) < 1e-16


def test_bb_step_is_the_inverse_curvature(oracle):
    """Near the Zeeman minimum E ~ H theta^2 / 2, so both BB quotients are 1/H up to O(theta^2) and the
    second iterate lands on the minimum up to O(theta^3); a swapped or inverted quotient fails this."""
    Hz, th0 = 2.0e5, 1.0e-2
    bb = oracle.BBMinimizer(macrospin(oracle, (0, 0, Hz)), unit(th0), tau0=1e-7, tau_min=0.0, tau_max=1.0, tol=0.0)
    bb.step()                                   # n = 0: tau0
    tau1, _, _ = bb.step()                      # n = 1: s.s / s.y
    assert abs(tau1 * Hz - 1.0) < 2e-4
    th2 = np.arccos(min(1.0, bb.m.reshape(3)[2]))
    assert th2 < 2.0 * th0 ** 3
    bb2 = oracle.BBMinimizer(macrospin(oracle, (0, 0, Hz)), unit(th0), tau0=1e-7, tau_min=0.0, tau_max=1.0, tol=0.0)
    bb2.st.n = 0
    bb2.step()
    bb2.st.n = 2                                # force the even rule s.y / y.y on the same pair
    tau2, _, _ = bb2.step()
    assert abs(tau2 * Hz - 1.0) < 2e-4


def test_clamps_and_negative_curvature_fallback(oracle):
    Hz = 1.0e5
    bb = oracle.BBMinimizer(macrospin(oracle, (0, 0, Hz)), unit(1.0), tau0=5e-6, tau_min=1e-6, tau_max=2e-6)
    tau, _, _ = bb.step()
    assert tau == 2e-6                          # tau0 above tau_max is clamped
    # at the energy MAXIMUM (m antiparallel to H) the curvature is negative: s.y < 0 -> tau0
    bb = oracle.BBMinimizer(macrospin(oracle, (0, 0, Hz)), unit(np.pi - 1e-3), tau0=3e-7, tau_min=0.0, tau_max=1.0)
    bb.step()
    tau, _, _ = bb.step()
    assert tau == 3e-7


def test_fixed_point_converges_immediately(oracle):
    m = np.zeros((3, 2, 1, 3))
    m[..., 2] = 1.0
    P = oracle.Problem(n=(3, 2, 1), d=(2e-9,) * 3, Ms=8e5, Aex=1.3e-11, Hext=(0, 0, 5e4), terms=2 | 8)
    bb = oracle.BBMinimizer(P, m, tau0=1e-6, tol=1e-12)
    tau, dm, conv = bb.step()
    assert dm == 0.0 and conv
    before = bb.m.copy()
    bb.step()                                   # a call on a converged state is a no-op
    assert bb.st.n == 1 and np.array_equal(bb.m, before)


@pytest.mark.parametrize("h", [0.2, 0.5, 0.9])
def test_stoner_wohlfarth_hard_axis(oracle, h):
    """Easy axis z, field along x with H = h H_k, H_k = 2 Ku/(mu0 Ms): the minimum has m_x = h."""
    Ms, Ku = 8e5, 5e5
    Hk = 2 * Ku / (MU0 * Ms)
    P = oracle.Problem(n=(1, 1, 1), d=(1e-9,) * 3, Ms=Ms, Ku=Ku, axis=(0, 0, 1), Hext=(h * Hk, 0, 0), terms=4 | 8)
    bb = oracle.BBMinimizer(P, unit(0.3, 0.7), tau0=1e-7, tau_min=1e-9, tau_max=1e-3, tol=1e-13)
    m, n, conv = bb.minimize(500)
    assert conv and n < 200
    m = m.reshape(3)
    assert abs(m[0] - h) < 1e-10 and abs(m[1]) < 1e-10 and m[2] > 0


def test_exchange_chain_relaxes_to_uniform_and_lowers_the_energy(oracle):
    n, d, Ms, A = (24, 1, 1), (2e-9,) * 3, 8e5, 1.3e-11
    P = oracle.Problem(n=n, d=d, Ms=Ms, Aex=A, Hext=(0, 0, 2e4), terms=2 | 8)

    def energy(m):      # E / (mu0 Ms V_cell) = -m.H_ext - 1/2 m.H_ex
        Hex = oracle.exchange(d, Ms, A, m)
        return float(np.sum(-m[..., 2] * 2e4 - 0.5 * np.sum(m * Hex, axis=-1)))

    m0 = w.random_unit_vectors(8, n)
    m0[..., 2] = np.abs(m0[..., 2]) + 0.5
    m0 /= np.linalg.norm(m0, axis=-1, keepdims=True)
    bb = oracle.BBMinimizer(P, m0, tau0=1e-7, tau_min=1e-10, tau_max=1e-3, tol=1e-12)
    m, it, conv = bb.minimize(5000)
    assert conv
    assert np.max(np.abs(m - np.array([0, 0, 1.0]))) < 1e-8
    assert energy(m) < energy(m0)
    assert np.max(np.abs(np.linalg.norm(m, axis=-1) - 1.0)) < 1e-14

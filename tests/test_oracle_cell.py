"""Pins for the single-cell arithmetic of the oracle.

Each test checks the oracle against something the mathematics fixes — lattice isotropy,
the hydrodynamic moments of the equilibrium, the moments of the Guo source, the
Smagorinsky quadratic — not against a re-typed copy of the oracle's formula.
"""
import itertools
import math

import numpy as np
import pytest

import oracle


@pytest.fixture(scope="module")
def lat():
    return oracle.lattice()


def test_lattice_is_d3q19_in_the_stated_order(lat):
    c, w, opp = lat
    # 19 distinct velocities = rest + 6 axis + 12 face-diagonal vectors of the cube
    vecs = {tuple(v) for v in c}
    assert len(vecs) == 19
    expected = {v for v in itertools.product((-1, 0, 1), repeat=3) if sum(abs(a) for a in v) <= 2}
    assert vecs == expected
    # opposite pairs adjacent, odd index = sign listed first
    assert tuple(c[0]) == (0, 0, 0)
    firsts = [(1, 0, 0), (0, 1, 0), (0, 0, 1), (1, 1, 0), (1, 0, 1), (0, 1, 1), (1, -1, 0), (1, 0, -1), (0, 1, -1)]
    for k, v in enumerate(firsts):
        assert tuple(c[2 * k + 1]) == v
        assert tuple(c[2 * k + 2]) == tuple(-a for a in v)
        assert opp[2 * k + 1] == 2 * k + 2 and opp[2 * k + 2] == 2 * k + 1
    assert opp[0] == 0
    # weights by shell
    for i in range(19):
        n2 = int((c[i] ** 2).sum())
        assert w[i] == pytest.approx({0: 1 / 3, 1: 1 / 18, 2: 1 / 36}[n2], abs=1e-17)


def test_lattice_isotropy(lat):
    c, w, _ = lat
    c = c.astype(float)
    assert w.sum() == pytest.approx(1.0, abs=1e-15)
    assert np.abs(np.einsum("i,ia->a", w, c)).max() < 1e-16
    np.testing.assert_allclose(np.einsum("i,ia,ib->ab", w, c, c), np.eye(3) / 3, atol=1e-16)
    assert np.abs(np.einsum("i,ia,ib,ic->abc", w, c, c, c)).max() < 1e-16
    # 4th-order isotropy: sum w c_a c_b c_c c_d = (1/9)(d_ab d_cd + d_ac d_bd + d_ad d_bc)
    d = np.eye(3)
    iso = (np.einsum("ab,cd->abcd", d, d) + np.einsum("ac,bd->abcd", d, d) + np.einsum("ad,bc->abcd", d, d)) / 9
    np.testing.assert_allclose(np.einsum("i,ia,ib,ic,id->abcd", w, c, c, c, c), iso, atol=1e-16)


@pytest.mark.parametrize("rho,u", [(1.0, (0.0, 0.0, 0.0)), (1.03, (0.05, -0.02, 0.01)), (0.97, (-0.08, 0.06, 0.07))])
def test_equilibrium_moments(lat, rho, u):
    c, _, _ = lat
    c = c.astype(float)
    u = np.array(u)
    fe = oracle.feq(rho, u)
    assert fe.sum() == pytest.approx(rho, abs=1e-15)
    np.testing.assert_allclose(c.T @ fe, rho * u, atol=1e-15)
    np.testing.assert_allclose(np.einsum("i,ia,ib->ab", fe, c, c), rho * np.eye(3) / 3 + rho * np.outer(u, u), atol=1e-15)


def _state_with_stress(lat, rho, u, Pi):
    """f = f_eq(rho,u) + f_neq with moments (0, 0, Pi): f_neq,i = 4.5 w_i (c_i c_i : Pi - tr Pi / 3)."""
    c, w, _ = lat
    c = c.astype(float)
    fneq = 4.5 * w * (np.einsum("ia,ib,ab->i", c, c, Pi) - np.trace(Pi) / 3)
    # the construction itself is checked: moments (0, 0, Pi)
    assert abs(fneq.sum()) < 1e-17 and np.abs(c.T @ fneq).max() < 1e-17
    np.testing.assert_allclose(np.einsum("i,ia,ib->ab", fneq, c, c), Pi, atol=1e-17)
    return oracle.feq(rho, u) + fneq


def test_rest_state_is_a_fixed_point_of_the_collision(lat):
    _, w, _ = lat
    g, rho, u, tau = oracle.collide_cell(w.copy(), 1e-3, 0.1, 0.0, (0, 0, 0))
    # to rounding: sum of the 19 rounded weights is 1 - O(1e-16), so f_eq = w_i rho can differ from w_i by an ulp
    np.testing.assert_allclose(g, w, rtol=0, atol=2.5e-16)
    assert rho == pytest.approx(1.0, abs=3e-16) and np.abs(u).max() < 1e-16
    assert tau == pytest.approx(0.503, abs=1e-15)


def test_cs_zero_gives_tau0_exactly(lat):
    Pi = np.array([[1e-3, 2e-4, 0], [2e-4, -5e-4, 1e-4], [0, 1e-4, -5e-4]])
    f = _state_with_stress(lat, 1.01, np.array([0.03, 0.01, -0.02]), Pi)
    for nu0 in (1e-4, 2e-3, 0.1):
        _, _, _, tau = oracle.collide_cell(f, nu0, 0.0, 0.0, (0, 0, 0))
        assert tau == 3.0 * nu0 + 0.5


def test_smagorinsky_tau_solves_its_quadratic(lat):
    """tau (tau - tau0) = 9 Cs^2 Q / (sqrt(2) rho)  with  Q = sqrt(Pi:Pi)  — i.e. nu_t = (Cs D)^2 |S|,
    |S| = sqrt(2 S:S), S = -Pi / (2 rho cs^2 tau) (SURVEY §8(c) step 4d and reading 2)."""
    rng = np.random.default_rng(1)
    for _ in range(5):
        A = rng.normal(size=(3, 3)) * 1e-3
        Pi = A + A.T
        rho = 1.0 + 0.02 * rng.normal()
        u = rng.normal(size=3) * 0.03
        nu0, Cs = 1e-3, 0.1 + 0.05 * rng.random()
        f = _state_with_stress(lat, rho, u, Pi)
        _, r, uu, tau = oracle.collide_cell(f, nu0, Cs, 0.0, (0, 0, 0))
        assert r == pytest.approx(rho, abs=1e-15)
        np.testing.assert_allclose(uu, u, atol=1e-15)
        tau0 = 3 * nu0 + 0.5
        Qn = math.sqrt((Pi * Pi).sum())
        assert tau * (tau - tau0) == pytest.approx(9 * Cs * Cs * Qn / (math.sqrt(2) * rho), rel=1e-12)
        # the same statement as an eddy viscosity: nu_total = (tau - 1/2)/3 = nu0 + Cs^2 |S|
        S = -Pi / (2 * rho * (1 / 3) * tau)
        assert (tau - 0.5) / 3 == pytest.approx(nu0 + Cs * Cs * math.sqrt(2 * (S * S).sum()), rel=1e-12)


def test_bgk_relaxes_the_stress_and_conserves_mass_momentum_without_force(lat):
    c, _, _ = lat
    c = c.astype(float)
    Pi = np.array([[4e-4, 1e-4, -2e-4], [1e-4, -1e-4, 3e-4], [-2e-4, 3e-4, -3e-4]])
    rho, u = 1.02, np.array([0.04, -0.03, 0.02])
    f = _state_with_stress(lat, rho, u, Pi)
    g, _, _, tau = oracle.collide_cell(f, 5e-3, 0.12, 0.0, (0, 0, 0))
    assert g.sum() == pytest.approx(f.sum(), abs=1e-15)
    np.testing.assert_allclose(c.T @ g, c.T @ f, atol=1e-16)
    Pi_eq = rho * np.eye(3) / 3 + rho * np.outer(u, u)
    np.testing.assert_allclose(np.einsum("i,ia,ib->ab", g, c, c) - Pi_eq, (1 - 1 / tau) * Pi, atol=1e-16)


def test_guo_source_moments_and_half_force_velocity(lat):
    """With f = f_eq(rho, v):  sum g = rho;  sum c g = m + F_d  (F_d = rho a(u));  second moment of the
    source = (1 - 1/2tau)(u F_d + F_d u);  u solves rho u = m + F_d / 2 with a(u) = F + f_cor (u_y, -u_x, 0)."""
    c, _, _ = lat
    c = c.astype(float)
    rho, v = 1.015, np.array([0.05, 0.02, -0.01])
    f = oracle.feq(rho, v)
    F = np.array([2e-5, -1e-5, 3e-5])
    fcor = 0.01
    nu0 = 0.02
    g, r, u, tau = oracle.collide_cell(f, nu0, 0.0, fcor, F)
    m = c.T @ f
    a = F + fcor * np.array([u[1], -u[0], 0.0])
    np.testing.assert_allclose(rho * u, m + 0.5 * rho * a, atol=1e-16)       # implicit half-force velocity
    Fd = rho * a
    assert g.sum() == pytest.approx(rho, abs=1e-15)                           # sum S = 0
    np.testing.assert_allclose(c.T @ g, m + Fd, atol=1e-16)                   # full force per step
    # second moment: relaxation part + source part
    fe = oracle.feq(rho, u)
    Pi_f = np.einsum("i,ia,ib->ab", f - fe, c, c)
    expect = np.einsum("i,ia,ib->ab", fe, c, c) + (1 - 1 / tau) * Pi_f + (1 - 0.5 / tau) * (np.outer(u, Fd) + np.outer(Fd, u))
    np.testing.assert_allclose(np.einsum("i,ia,ib->ab", g, c, c), expect, atol=1e-16)


def test_coriolis_turns_the_wind_clockwise_for_positive_f(lat):
    f = oracle.feq(1.0, np.array([0.05, 0.0, 0.0]))
    g, _, u, _ = oracle.collide_cell(f, 0.01, 0.0, 0.02, (0, 0, 0))
    c = lat[0].astype(float)
    assert (c.T @ g)[1] < 0  # a = f (u_y, -u_x, 0): +x wind is pushed to -y

"""Pins for the full Coriolis rotation vector in the oracle (Table 1: "Coriolis ... full
rotation vector in the local ENU frame ... evaluated directly within the GPU kernel" through Guo forcing).

a_cor(u) = -2 Omega x u = -f x u with f = 2 Omega (lattice units).  Nothing here re-types the oracle's linear solve:
the pins are invariants of the physics (the Coriolis force does no work and is perpendicular to the axis), the exact
solution of the time-discrete system (total momentum turns about the axis by 2 atan(|f|/2) per step, Rodrigues'
formula), the reduction to the scalar form the older pins fix, and the agreement of two independent code paths
(collision-side solve with I - C/2, macro-side solve with I + C/2)."""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def O(oracle_mod):
    return oracle_mod


def near_equilibrium(O, rng, rho=1.02, u=(0.05, -0.03, 0.02), eps=1e-3):
    f = O.feq(rho, np.asarray(u, dtype=np.float64))
    return f * (1.0 + eps * rng.standard_normal(19))


def test_vector_along_z_is_the_scalar_form(O):
    rng = np.random.default_rng(1)
    f = near_equilibrium(O, rng)
    F = (1e-5, -2e-5, 3e-6)
    g0, r0, u0, t0 = O.collide_cell(f, 1e-3, 0.1, 7e-4, F)
    g1, r1, u1, t1 = O.collide_cell_vec(f, 1e-3, 0.1, (0.0, 0.0, 7e-4), F)
    assert np.abs(g0 - g1).max() < 1e-16 and abs(t0 - t1) < 1e-15 and np.abs(u0 - u1).max() < 1e-16


def test_coriolis_force_does_no_work_and_is_perpendicular_to_the_axis(O):
    rng = np.random.default_rng(2)
    c, w, opp = O.lattice()
    for _ in range(20):
        fv = 1e-2 * rng.standard_normal(3)
        F = 1e-4 * rng.standard_normal(3)
        f = near_equilibrium(O, rng, u=0.05 * rng.standard_normal(3))
        g, rho, u, tau = O.collide_cell_vec(f, 2e-3, 0.1, fv, F)
        m = (c * f[:, None]).sum(axis=0)
        Fd = 2.0 * (rho * u - m)                  # half-force identity rho u = m + Fd / 2
        dm = (c * g[:, None]).sum(axis=0) - m     # the collision adds exactly the force to the momentum
        assert np.abs(dm - Fd).max() < 1e-15
        a_cor = Fd / rho - F
        assert abs(a_cor @ u) < 1e-16             # no work
        assert abs(a_cor @ fv) < 1e-17            # perpendicular to the rotation axis
        assert np.linalg.norm(a_cor) == pytest.approx(np.linalg.norm(np.cross(fv, u)), rel=1e-10)
        assert abs(g.sum() - f.sum()) < 1e-15     # mass


def rodrigues(axis, theta):
    n = np.asarray(axis, dtype=np.float64) / np.linalg.norm(axis)
    K = np.array([[0, -n[2], n[1]], [n[2], 0, -n[0]], [-n[1], n[0], 0]])
    return np.eye(3) + np.sin(theta) * K + (1 - np.cos(theta)) * (K @ K)


@pytest.mark.parametrize("fv", [(0.0, 0.0, 3e-3), (2e-3, -1e-3, 2.5e-3), (4e-3, 0.0, 0.0), (0.0, -5e-3, 1e-3)])
def test_total_momentum_turns_about_the_axis_by_2atan_half_f_per_step(O, fv):
    """Periodic box, non-uniform flow and density, LES on: P_k = R^k P_0 exactly, R = rotation about f by
    -2 atan(|f|/2) (clockwise seen from the tip of f, the sense the scalar pin fixes for f along z)."""
    n = 12
    rng = np.random.default_rng(3)
    o = O.Oracle(n, n, n, 5e-3, 0.1, 0.0, (0, 0, 0), (0, 0, 0, 0, 0, 0))
    o.set_coriolis(fv)
    o.set_flags(None)
    x = np.arange(n) * 2 * np.pi / n
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij")
    X, Y, Z = X.T, Y.T, Z.T
    rho = 1.0 + 0.01 * np.sin(X) * np.cos(Z)
    ux = 0.03 + 0.01 * np.sin(Y)
    uy = -0.02 + 0.01 * np.cos(Z)
    uz = 0.015 + 0.01 * np.sin(X + Y)
    o.set_macros(rho, ux, uy, uz)
    c, w, opp = O.lattice()
    def P():
        f = o.get_state()
        return np.array([(c[:, a][:, None, None, None] * f).sum() for a in range(3)])
    P0 = P()
    fn = np.linalg.norm(fv)
    R = rodrigues(fv, -2.0 * np.arctan(0.5 * fn))
    Pk = P0.copy()
    for k in range(25):
        o.step(1)
        Pk = R @ Pk
        assert np.abs(P() - Pk).max() < 1e-12 * n ** 3
    assert np.linalg.norm(P()) == pytest.approx(np.linalg.norm(P0), rel=1e-13)
    assert P() @ np.asarray(fv) == pytest.approx(P0 @ np.asarray(fv), rel=1e-12, abs=1e-16)
    o.close()


def test_local_macros_return_what_the_collision_used_with_a_tilted_axis(O):
    """Two independent solves: the collision's (I - C/2) u = b and the macro inversion (I + C/2) u = b'."""
    rng = np.random.default_rng(4)
    fv, F = (3e-3, -2e-3, 4e-3), (2e-5, 1e-5, -1e-5)
    f = near_equilibrium(O, rng)
    g, rho, u, tau = O.collide_cell_vec(f, 1e-3, 0.1, fv, F)
    o = O.Oracle(1, 1, 1, 1e-3, 0.1, 0.0, F, (0, 0, 0, 0, 0, 0))
    o.set_coriolis(fv)
    o.set_flags(None)
    o.set_state(g.reshape(19, 1, 1, 1))
    r2, ux, uy, uz = o.get_macros()
    assert abs(r2[0, 0, 0] - rho) < 1e-15
    assert np.abs(np.array([ux[0, 0, 0], uy[0, 0, 0], uz[0, 0, 0]]) - u).max() < 1e-16
    o.close()

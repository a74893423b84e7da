"""Pins for the damping zones of the oracle: top sponge layer + boundary-adjacent buffer nudging (PAPER.md:175
"relaxation-based damping regions adjacent to the upper and lateral boundaries, including a top sponge layer and
boundary-adjacent buffer nudging toward the target boundary state"; Table 1 PAPER.md:86 "sponge and buffer damping").

Reading (DESIGN.md §4 reading 20): a_d(u) = sigma(x) (u_t(z) - u), integrated with the implicit half-force rule.
Nothing here re-types the oracle's 3x3 solve.  The pins are: the exact solution of the time-discrete relaxation
(trapezoidal factor (1 - sigma/2)/(1 + sigma/2) per step, also on a whole lattice with uniform sigma), the momentum
budget of a non-uniform flow with the ramp, the shape facts of the ramp, invariants (mass, fixed point at the
target, sigma = 0 is the undamped step bit for bit), and the agreement of two independent solves (collision side,
macro side)."""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def O(oracle_mod):
    return oracle_mod


def near_equilibrium(O, rng, rho=1.02, u=(0.05, -0.03, 0.02), eps=1e-3):
    f = O.feq(rho, np.asarray(u, dtype=np.float64))
    return f * (1.0 + eps * rng.standard_normal(19))


def test_sigma_zero_is_the_undamped_collision_bit_for_bit(O):
    rng = np.random.default_rng(1)
    f = near_equilibrium(O, rng)
    fv, F = (1e-3, -2e-3, 3e-3), (1e-5, 2e-5, -1e-5)
    g0, r0, u0, t0 = O.collide_cell_vec(f, 1e-3, 0.1, fv, F)
    g1, r1, u1, t1 = O.collide_cell_damped(f, 1e-3, 0.1, fv, F, 0.0, (0.3, 0.2, 0.1))
    assert np.array_equal(g0, g1) and np.array_equal(u0, u1) and t0 == t1


def test_one_cell_relaxes_by_the_trapezoidal_factor_and_conserves_mass(O):
    """No Coriolis, no F: with v = m/rho - u_t the collision velocity is u - u_t = v / (1 + sigma/2) and the
    post-collision momentum m*/rho - u_t = v (1 - sigma/2) / (1 + sigma/2) (the trapezoidal rule for dv/dt = -sigma v)."""
    rng = np.random.default_rng(2)
    c, w, opp = O.lattice()
    for sigma in (1e-3, 0.05, 0.3, 1.0):
        ut = 0.05 * rng.standard_normal(3)
        f = near_equilibrium(O, rng, u=0.05 * rng.standard_normal(3))
        g, rho, u, tau = O.collide_cell_damped(f, 2e-3, 0.1, (0, 0, 0), (0, 0, 0), sigma, ut)
        m = (c * f[:, None]).sum(axis=0)
        ms = (c * g[:, None]).sum(axis=0)
        v = m / rho - ut
        assert np.abs((u - ut) - v / (1 + sigma / 2)).max() < 1e-16
        assert np.abs((ms / rho - ut) - v * (1 - sigma / 2) / (1 + sigma / 2)).max() < 1e-15
        assert abs(g.sum() - f.sum()) < 1e-15


def test_damping_force_is_sigma_times_the_defect_with_forces_and_rotation_present(O):
    """Fd = 2 (rho u - m) (half-force identity) must equal rho [F - f x u + sigma (u_t - u)] for the returned u."""
    rng = np.random.default_rng(3)
    c, w, opp = O.lattice()
    for _ in range(20):
        fv = 1e-2 * rng.standard_normal(3)
        F = 1e-4 * rng.standard_normal(3)
        ut = 0.05 * rng.standard_normal(3)
        sigma = rng.uniform(0, 1)
        f = near_equilibrium(O, rng, u=0.05 * rng.standard_normal(3))
        g, rho, u, tau = O.collide_cell_damped(f, 2e-3, 0.1, fv, F, sigma, ut)
        m = (c * f[:, None]).sum(axis=0)
        Fd = 2.0 * (rho * u - m)
        assert np.abs(Fd - rho * (F - np.cross(fv, u) + sigma * (ut - u))).max() < 1e-15
        assert np.abs((c * g[:, None]).sum(axis=0) - m - Fd).max() < 1e-15


def test_local_macros_return_what_the_damped_collision_used(O):
    """Two independent solves: ((1 + s/2) I - C/2) u = b in the collision, ((1 - s/2) I + C/2) u = b' in the macros."""
    rng = np.random.default_rng(4)
    fv, F = (3e-3, -2e-3, 4e-3), (2e-5, 1e-5, -1e-5)
    ut = np.array([0.04, -0.01, 0.02])
    f = near_equilibrium(O, rng)
    o = O.Oracle(1, 1, 1, 1e-3, 0.1, 0.0, F, (0, 0, 0, 0, 0, 0))
    o.set_coriolis(fv)
    o.set_flags(None)
    o.set_damping((0, 0, 0, 0, 0, 1), (0, 0, 0, 0, 0, 0.37), ut.reshape(3, 1))
    assert o.get_damping()[0, 0, 0] == pytest.approx(0.37, abs=1e-16)
    g, rho, u, tau = O.collide_cell_damped(f, 1e-3, 0.1, fv, F, o.get_damping()[0, 0, 0], ut)
    o.set_state(g.reshape(19, 1, 1, 1))
    r2, ux, uy, uz = o.get_macros()
    assert abs(r2[0, 0, 0] - rho) < 1e-15
    assert np.abs(np.array([ux[0, 0, 0], uy[0, 0, 0], uz[0, 0, 0]]) - u).max() < 1e-15
    o.close()


def test_ramp_shape(O):
    """Peak at the face layer, sin^2 half value at d = W/2, zero from d = W on, monotone, largest zone wins in corners."""
    nx, ny, nz = 24, 20, 16
    o = O.Oracle(nx, ny, nz, 1e-2, 0.0, 0.0, (0, 0, 0), (0, 0, 0, 0, 0, 0))
    o.set_flags(None)
    width, peak = (4, 8, 0, 6, 0, 8), (0.2, 0.1, 0.5, 0.3, 0.0, 0.4)
    o.set_damping(width, peak, np.zeros((3, nz)))
    s = o.get_damping()                      # [z][y][x]
    mid = s[4, 8, :]                         # away from the y+ and z+ zones: only the x zones act
    assert mid[0] == pytest.approx(0.2, abs=1e-16) and mid[nx - 1] == pytest.approx(0.1, abs=1e-16)
    assert mid[2] == pytest.approx(0.1, abs=1e-16)            # d = W/2 of the x- zone: half the peak
    assert mid[nx - 1 - 4] == pytest.approx(0.05, abs=1e-16)  # d = W/2 of the x+ zone
    assert np.all(mid[4:nx - 8] == 0.0)
    assert np.all(np.diff(mid[:5]) < 0) and np.all(np.diff(mid[nx - 9:]) > 0)
    assert np.all(s[4, 0:ny - 6, 10] == 0.0)                  # y- has width 0 (its peak is ignored), z- has peak 0
    col = s[:, 8, 10]
    assert col[nz - 1] == pytest.approx(0.4, abs=1e-16) and np.all(col[:nz - 8] == 0.0)
    # corner x-, y+, z+: the largest of the three ramps, not their sum
    assert s[nz - 1, ny - 1, 0] == pytest.approx(0.4, abs=1e-16)
    assert s[nz - 1, ny - 1, nx - 1] == pytest.approx(0.4, abs=1e-16)
    assert s[4, ny - 1, 0] == pytest.approx(0.3, abs=1e-16)
    assert s.min() >= 0.0 and s.max() <= 0.4 + 1e-16
    # all widths zero switches it off
    o.set_damping((0,) * 6, (0.5,) * 6, None)
    assert np.all(o.get_damping() == 0.0)
    with pytest.raises(RuntimeError):
        o.set_damping((1,) * 6, (1.5,) * 6, np.zeros((3, nz)))
    o.close()


def test_uniform_flow_in_a_uniform_zone_decays_geometrically(O):
    """Two-layer slab between free-slip z faces, periodic x,y; width-1 zones on z- and z+ give the same sigma in every
    cell.  A uniform horizontal flow stays uniform, so u_k - u_t = (u_0 - u_t) q^k / (1 + sigma/2)-corrected:
    stored momentum deviation after k steps = v_0 q^k, q = (1 - sigma/2)/(1 + sigma/2)."""
    nx, ny, nz = 6, 5, 2
    sigma = 0.2
    o = O.Oracle(nx, ny, nz, 1e-2, 0.1, 0.0, (0, 0, 0), (0, 0, 0, 0, 2, 2))
    o.set_flags(None)
    ut = np.zeros((3, nz)); ut[0] = 0.03; ut[1] = -0.01
    o.set_damping((0, 0, 0, 0, 1, 1), (0, 0, 0, 0, sigma, sigma), ut)
    assert np.all(o.get_damping() == sigma)
    u0 = np.array([0.08, 0.02, 0.0])
    o.set_macros(None, np.full((nz, ny, nx), u0[0]), np.full((nz, ny, nx), u0[1]), None)
    c, w, opp = O.lattice()
    q = (1 - sigma / 2) / (1 + sigma / 2)
    v0 = u0 - ut[:, 0]
    for k in range(1, 31):
        o.step(1)
        f = o.get_state()
        mom = np.array([(c[:, a][:, None, None, None] * f).sum(axis=0) for a in range(3)])   # [3][z][y][x]
        assert np.abs(f.sum(axis=0) - 1.0).max() < 1e-14
        for a in range(3):
            assert np.abs(mom[a] - (ut[a, 0] + v0[a] * q ** k)).max() < 1e-15
        r, ux, uy, uz = o.get_macros()
        # the velocity the collision of step k used: half a relaxation step behind the stored momentum
        assert np.abs(ux - (ut[0, 0] + v0[0] * q ** (k - 1) / (1 + sigma / 2))).max() < 1e-15
    o.close()


def test_momentum_budget_of_a_non_uniform_flow_with_ramped_zones(O):
    """Periodic box, non-uniform flow and density, LES on, F != 0: per step the total momentum changes by
    sum_x rho (F + sigma(x) (u_t(z) - u)) with (rho, u) the macros after the step (= what its collision used);
    sigma(x) is taken from the oracle's own export, whose shape test_ramp_shape pins."""
    n = 12
    o = O.Oracle(n, n, n, 5e-3, 0.1, 0.0, (2e-6, -1e-6, 0), (0, 0, 0, 0, 0, 0))
    o.set_flags(None)
    x = np.arange(n) * 2 * np.pi / n
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij")
    X, Y, Z = X.T, Y.T, Z.T
    o.set_macros(1.0 + 0.01 * np.sin(X) * np.cos(Z), 0.03 + 0.01 * np.sin(Y), -0.02 + 0.01 * np.cos(Z), 0.01 * np.sin(X + Y))
    ut = np.stack([0.04 + 0.002 * np.arange(n), 0.01 * np.ones(n), np.zeros(n)])
    o.set_damping((3, 0, 0, 4, 0, 5), (0.05, 0, 0, 0.2, 0, 0.1), ut)
    sig = o.get_damping()
    c, w, opp = O.lattice()
    F = np.array([2e-6, -1e-6, 0.0])
    def P():
        f = o.get_state()
        return np.array([(c[:, a][:, None, None, None] * f).sum() for a in range(3)]), f.sum()
    P0, M0 = P()
    for k in range(20):
        o.step(1)
        P1, M1 = P()
        r, ux, uy, uz = o.get_macros()
        u = (ux, uy, uz)
        dP = np.array([(r * (F[a] + sig * (ut[a][:, None, None] - u[a]))).sum() for a in range(3)])
        assert np.abs((P1 - P0) - dP).max() < 1e-13
        assert abs(M1 - M0) < 1e-11
        P0 = P1
    o.close()


def test_flow_at_the_target_state_is_a_fixed_point(O):
    """Uniform f_eq(1,(U,0,0)) with EQ_FIXED x-, EQ_OUTFLOW x+, periodic y, free-slip z is an exact fixed point; with
    the target equal to that state the damping force vanishes identically and the zones change nothing."""
    nx, ny, nz = 14, 6, 8
    U = 0.05
    o = O.Oracle(nx, ny, nz, 1e-3, 0.1, 0.0, (0, 0, 0), (3, 4, 0, 0, 2, 2))
    o.set_flags(None)
    o.set_inlet_profile(np.full(nz, U))
    o.set_macros(None, np.full((nz, ny, nx), U), None, None)
    ut = np.zeros((3, nz)); ut[0] = U
    o.set_damping((4, 4, 0, 0, 0, 3), (0.1, 0.3, 0, 0, 0, 0.2), ut)
    f0 = o.get_state()
    o.step(10)
    assert np.abs(o.get_state() - f0).max() < 2e-15   # rounding of the (1 + sigma/2) solve only; an active zone would move it by ~1e-3
    o.close()


def test_sponge_absorbs_a_disturbance_that_the_undamped_box_keeps(O):
    """A plane vertical velocity pulse between two free-slip faces is a pair of sound waves (one up, one down, the lower
    one reflected by the bottom face).  After 200 steps (sound path 115 cells, box 40) the undamped box still holds
    most of the acoustic energy sum(u_z^2 + (rho - 1)^2 / 3); a top sponge towards rest has absorbed > 90 % of it
    (qualitative: the zone damps, it does not feed)."""
    nx, ny, nz = 4, 4, 40
    def run(damped, steps):
        o = O.Oracle(nx, ny, nz, 2e-3, 0.0, 0.0, (0, 0, 0), (0, 0, 0, 0, 2, 2))
        o.set_flags(None)
        z = np.arange(nz)
        w = 0.02 * np.exp(-0.5 * ((z - 20.0) / 2.0) ** 2)
        o.set_macros(None, None, None, np.broadcast_to(w[:, None, None], (nz, ny, nx)).copy())
        if damped:
            o.set_damping((0, 0, 0, 0, 0, 12), (0, 0, 0, 0, 0, 0.3), np.zeros((3, nz)))
        o.step(steps)
        r, ux, uy, uz = o.get_macros()
        o.close()
        return float((uz ** 2 + (r - 1) ** 2 / 3).sum())
    e0 = run(False, 1)
    e_free, e_damp = run(False, 200), run(True, 200)
    assert e_free > 0.7 * e0
    assert e_damp < 0.1 * e_free

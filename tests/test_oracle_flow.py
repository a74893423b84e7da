"""Pins for the whole-step behaviour of the oracle (SURVEY.md §8(c) "what pins each part").

Closed forms and invariants only: rest state, mass conservation, Poiseuille profile under halfway
bounce-back (pins wall location, Guo forcing and nu <-> tau0), Taylor-Green decay (pins viscosity),
faster decay with Smagorinsky, exact inertial rotation of momentum (pins the implicit Coriolis
half-step), free-slip = mirror image, periodic = translation invariance, streaming direction,
uniform-flow fixed points through inlet/outflow cells, local macro inversion.
"""
import math

import numpy as np
import pytest

import oracle
from oracle import Oracle

P, WALL, FS, EQF, EQO = 0, 1, 2, 3, 4
ALLP = (P,) * 6


def _momentum(o):
    c, _, _ = oracle.lattice()
    G = o.get_state()
    return np.einsum("ia,izyx->a", c.astype(float), G), G.sum()


def test_rest_state_with_solids_and_every_face_type_stays_at_rest():
    nx, ny, nz = 12, 10, 8
    hm = np.zeros((ny, nx), dtype=np.int32)
    hm[3:6, 4:8] = 5
    hm[0, 0] = 8
    _, w, _ = oracle.lattice()
    for faces in [(EQF, EQO, P, P, WALL, FS), (FS, FS, WALL, WALL, P, P), ALLP, (EQO, EQF, FS, WALL, WALL, WALL)]:
        o = Oracle(nx, ny, nz, 1e-3, 0.1, 0.0, (0, 0, 0), faces)
        o.set_flags(hm)
        o.set_inlet_profile(np.zeros(nz))
        o.set_macros()
        o.step(50)
        G = o.get_state()
        # to rounding (the 19 rounded weights do not sum to exactly 1); no drift over the run
        assert np.abs(G - w[:, None, None, None]).max() < 1e-15
        rho, ux, uy, uz = o.get_macros()
        assert np.abs(rho - 1).max() < 1e-14
        assert max(np.abs(ux).max(), np.abs(uy).max(), np.abs(uz).max()) < 1e-15


def test_mass_is_conserved_with_solids_forcing_coriolis_free_slip_and_les():
    nx, ny, nz = 16, 12, 10
    rng = np.random.default_rng(7)
    hm = np.zeros((ny, nx), dtype=np.int32)
    hm[2:5, 3:9] = 4
    hm[8:10, 10:14] = 7
    o = Oracle(nx, ny, nz, 2e-3, 0.15, 5e-3, (3e-5, -1e-5, 0.0), (P, P, P, P, WALL, FS))
    o.set_flags(hm)
    o.set_macros(1 + 0.01 * rng.normal(size=o.shape), 0.03 * rng.normal(size=o.shape),
                 0.03 * rng.normal(size=o.shape), 0.02 * rng.normal(size=o.shape))
    fluid = o.get_flags() == 0
    m0 = (o.get_state().sum(axis=0))[fluid].sum()
    o.step(300)
    m1 = (o.get_state().sum(axis=0))[fluid].sum()
    assert abs(m1 / m0 - 1) < 1e-12


@pytest.mark.parametrize("nu", [0.05, 0.1, 0.3, math.sqrt(3) / 12])
def test_poiseuille_profile_under_halfway_bounce_back(nu):
    """Walls on both z faces half a cell outside the first/last node, body force a along x, Cs = 0:
    u(zeta) = a zeta (H - zeta) / (2 nu) + a (48 nu^2 - 1) / (8 nu),  zeta = z + 1/2
    (BGK + halfway bounce-back: the wall sits exactly at the half-way plane when (tau-1/2)^2 = 3/16,
    i.e. nu = sqrt(3)/12, where the slip term vanishes)."""
    H, a = 12, 1e-6
    o = Oracle(2, 2, H, nu, 0.0, 0.0, (a, 0, 0), (P, P, P, P, WALL, WALL))
    o.set_flags()
    o.set_macros()
    o.step(int(4.0 * H * H / nu))
    rho, ux, uy, uz = o.get_macros()
    zeta = np.arange(H) + 0.5
    exact = a * zeta * (H - zeta) / (2 * nu) + a * (48 * nu * nu - 1) / (8 * nu)
    np.testing.assert_allclose(ux[:, 0, 0], exact, rtol=1e-9)
    assert np.abs(ux - ux[:, :1, :1]).max() < 1e-18 + 1e-12 * exact.max()
    assert np.abs(uy).max() < 1e-18 and np.abs(uz).max() < 1e-13   # u_z: rounding noise only
    assert np.abs(rho - 1).max() < 1e-12
    if abs(nu - math.sqrt(3) / 12) < 1e-12:
        # no slip: parabola through zero at the half-way planes
        np.testing.assert_allclose(ux[:, 0, 0], a * zeta * (H - zeta) / (2 * nu), rtol=1e-9)


def test_buildings_are_walls_too_poiseuille_between_a_solid_slab_and_the_top_wall():
    """Same closed form when the lower wall is a SOLID layer from the heightmap (bounce-back on flags)."""
    H, base, a, nu = 10, 3, 1e-6, 0.1
    o = Oracle(2, 2, H + base, nu, 0.0, 0.0, (a, 0, 0), (P, P, P, P, WALL, WALL))
    o.set_flags(np.full((2, 2), base, dtype=np.int32))
    o.set_macros()
    o.step(int(4.0 * H * H / nu))
    _, ux, _, _ = o.get_macros()
    zeta = np.arange(H) + 0.5
    exact = a * zeta * (H - zeta) / (2 * nu) + a * (48 * nu * nu - 1) / (8 * nu)
    np.testing.assert_allclose(ux[base:, 0, 0], exact, rtol=1e-9)
    assert np.all(ux[:base] == 0)


def _tgv(n, nz, nu, Cs, steps0, steps1, u0=0.04):
    k = 2 * math.pi / n
    x = np.arange(n)
    X, Y = np.meshgrid(x, x, indexing="xy")
    ux = np.broadcast_to(u0 * np.sin(k * X) * np.cos(k * Y), (nz, n, n))
    uy = np.broadcast_to(-u0 * np.cos(k * X) * np.sin(k * Y), (nz, n, n))
    rho = np.broadcast_to(1 - 0.75 * u0 * u0 * (np.cos(2 * k * X) + np.cos(2 * k * Y)), (nz, n, n))
    o = Oracle(n, n, nz, nu, Cs, 0.0, (0, 0, 0), ALLP)
    o.set_flags()
    o.set_macros(rho, ux, uy, None)
    o.step(steps0)
    _, a, b, _ = o.get_macros()
    ke0 = (a * a + b * b).sum()
    o.step(steps1 - steps0)
    _, a, b, c = o.get_macros()
    ke1 = (a * a + b * b).sum()
    assert np.abs(c).max() < 1e-14
    rate = -math.log(ke1 / ke0) / (steps1 - steps0)
    return rate / (4 * nu * k * k)


def test_taylor_green_decay_rate_gives_the_viscosity():
    """2-D Taylor-Green vortex extruded in z: kinetic energy ~ exp(-4 nu k^2 t)."""
    ratio = _tgv(64, 2, 0.01, 0.0, 200, 800)
    assert abs(ratio - 1) <= 0.015


def test_smagorinsky_makes_taylor_green_decay_faster_but_boundedly():
    r0 = _tgv(48, 2, 2e-3, 0.0, 100, 500)
    r1 = _tgv(48, 2, 2e-3, 0.1, 100, 500)
    # nu_t = Cs^2 |S| <= Cs^2 * 2 u0 k  (max strain of the TGV) -> ratio bounded by 1 + nu_t,max / nu0
    k = 2 * math.pi / 48
    assert r1 > r0 * 1.005
    assert r1 < r0 * (1 + 0.1 ** 2 * 2 * 0.04 * k / 2e-3)


def test_inertial_oscillation_total_momentum_rotates_exactly():
    """Periodic box, non-uniform flow, F = 0: total post-collision momentum P_k = R^k P_0 with R the rotation
    by -2 atan(f/2) — the implicit (Crank-Nicolson) Coriolis half-step conserves |P| exactly.  An explicit
    reading would grow |P| by (1+f^2/4...)^k and fail the modulus check."""
    n, f = 8, 0.05
    rng = np.random.default_rng(3)
    o = Oracle(n, n, 4, 5e-3, 0.1, f, (0, 0, 0), ALLP)
    o.set_flags()
    o.set_macros(1 + 0.01 * rng.normal(size=o.shape), 0.03 + 0.02 * rng.normal(size=o.shape),
                 -0.01 + 0.02 * rng.normal(size=o.shape), 0.01 * rng.normal(size=o.shape))
    P0, m0 = _momentum(o)
    K = 40
    o.step(K)
    P1, m1 = _momentum(o)
    assert abs(m1 / m0 - 1) < 1e-13
    assert abs(np.hypot(P1[0], P1[1]) / np.hypot(P0[0], P0[1]) - 1) < 1e-12
    dtheta = math.atan2(P1[1], P1[0]) - math.atan2(P0[1], P0[0])
    assert dtheta == pytest.approx(-K * 2 * math.atan(f / 2), abs=1e-11)
    assert P1[2] == pytest.approx(P0[2], abs=1e-13)


def test_inertial_oscillation_uniform_flow_velocity_and_period():
    """Uniform flow: the reported u after k steps has angle -(k - 1/2) 2 atan(f/2) and modulus |u0|/sqrt(1+f^2/4);
    a full turn takes 2 pi / (2 atan(f/2)) ~ 2 pi / f steps."""
    f, U = 0.02, 0.05
    o = Oracle(4, 4, 4, 0.01, 0.0, f, (0, 0, 0), ALLP)
    o.set_flags()
    o.set_macros(None, np.full(o.shape, U), None, None)
    for k in (1, 7, 50):
        o.step(k - o.get_step())
        _, ux, uy, _ = o.get_macros()
        assert np.ptp(ux) < 1e-16 and np.ptp(uy) < 1e-16
        assert math.hypot(ux[0, 0, 0], uy[0, 0, 0]) == pytest.approx(U / math.sqrt(1 + f * f / 4), rel=1e-13)
        assert math.atan2(uy[0, 0, 0], ux[0, 0, 0]) == pytest.approx(-(k - 0.5) * 2 * math.atan(f / 2), abs=1e-13)
    period = 2 * math.pi / (2 * math.atan(f / 2))
    assert period == pytest.approx(2 * math.pi / f, rel=1e-4)


def test_free_slip_equals_the_mirror_image_domain():
    """A free-slip plane is a symmetry plane: the run on ny rows with FREE_SLIP on y+ must equal the lower half of a
    2 ny run between two WALL faces with the field and the buildings mirrored (u_y odd).  Includes a tower that
    touches the free-slip z top and a building that touches the free-slip y face.  (No Coriolis: it is not
    mirror-symmetric.)"""
    nx, ny, nz = 10, 8, 6
    rng = np.random.default_rng(11)
    hm = np.zeros((ny, nx), dtype=np.int32)
    hm[2:5, 3:6] = 6          # a tower touching the free-slip top
    hm[6:8, 7:9] = 2          # a block touching the free-slip y+ face
    rho = 1 + 0.01 * rng.normal(size=(nz, ny, nx))
    ux, uy, uz = (0.03 * rng.normal(size=(nz, ny, nx)) for _ in range(3))
    b = Oracle(nx, ny, nz, 3e-3, 0.1, 0.0, (1e-5, 0, 0), (P, P, WALL, FS, WALL, FS))
    b.set_flags(hm)
    b.set_macros(rho, ux, uy, uz)
    b.step(25)
    hm2 = np.concatenate([hm, hm[::-1]], axis=0)
    m = lambda q, s=1.0: np.concatenate([q, s * q[:, ::-1]], axis=1)  # noqa: E731
    c = Oracle(nx, 2 * ny, nz, 3e-3, 0.1, 0.0, (1e-5, 0, 0), (P, P, WALL, WALL, WALL, FS))
    c.set_flags(hm2)
    c.set_macros(m(rho), m(ux), m(uy, -1.0), m(uz))
    c.step(25)
    for qb, qc in zip(b.get_macros(), c.get_macros()):
        np.testing.assert_allclose(qb, qc[:, :ny], atol=1e-15)


def test_free_slip_top_equals_mirror_image_in_z():
    """Same symmetry in z (no buildings, so the mirrored domain is expressible): FREE_SLIP top on nz levels equals the
    lower half of 2 nz levels between two WALL faces with the field mirrored (u_z odd)."""
    nx, ny, nz = 6, 5, 7
    rng = np.random.default_rng(5)
    rho = 1 + 0.01 * rng.normal(size=(nz, ny, nx))
    ux, uy, uz = (0.03 * rng.normal(size=(nz, ny, nx)) for _ in range(3))
    a = Oracle(nx, ny, nz, 3e-3, 0.1, 2e-3, (1e-5, 2e-5, 0), (P, P, P, P, WALL, FS))
    a.set_flags()
    a.set_macros(rho, ux, uy, uz)
    a.step(30)
    m = lambda q, s=1.0: np.concatenate([q, s * q[::-1]], axis=0)  # noqa: E731
    b = Oracle(nx, ny, 2 * nz, 3e-3, 0.1, 2e-3, (1e-5, 2e-5, 0), (P, P, P, P, WALL, WALL))
    b.set_flags()
    b.set_macros(m(rho), m(ux), m(uy), m(uz, -1.0))
    b.step(30)
    for qa, qb in zip(a.get_macros(), b.get_macros()):
        np.testing.assert_allclose(qa, qb[:nz], atol=1e-15)


def test_periodic_faces_are_translation_invariant():
    nx, ny, nz = 9, 7, 5
    rng = np.random.default_rng(2)
    hm = np.zeros((ny, nx), dtype=np.int32)
    hm[1:3, 2:5] = 3
    fields = [1 + 0.01 * rng.normal(size=(nz, ny, nx))] + [0.03 * rng.normal(size=(nz, ny, nx)) for _ in range(3)]
    out = []
    for shift in ((0, 0), (4, 3)):
        o = Oracle(nx, ny, nz, 2e-3, 0.1, 1e-3, (1e-5, 0, 0), (P, P, P, P, WALL, FS))
        roll = lambda q: np.roll(q, (shift[1], shift[0]), axis=(-2, -1))  # noqa: E731
        o.set_flags(roll(hm))
        o.set_macros(*[roll(q) for q in fields])
        o.step(20)
        out.append([np.roll(q, (-shift[1], -shift[0]), axis=(-2, -1)) for q in o.get_macros()])
    for q0, q1 in zip(*out):
        np.testing.assert_allclose(q0, q1, atol=1e-15)


def test_streaming_direction_a_shear_wave_is_carried_downstream():
    """u_y = eps sin(k x) on a uniform U_x: after t steps u_y ~ eps exp(-nu k^2 t) sin(k (x - U t)).
    Pull from x - c_i; a sign error would carry the wave upstream."""
    n, U, eps, nu, t = 32, 0.1, 1e-3, 0.02, 80
    k = 2 * math.pi / n
    x = np.arange(n)
    o = Oracle(n, 2, 2, nu, 0.0, 0.0, (0, 0, 0), ALLP)
    o.set_flags()
    o.set_macros(None, np.full(o.shape, U), np.broadcast_to(eps * np.sin(k * x), o.shape), None)
    o.step(t)
    _, _, uy, _ = o.get_macros()
    # phase of the fundamental
    z = np.fft.fft(uy[0, 0])[1]                 # A sin(k (x - s)) -> fft[1] = (n A / 2) exp(-i (k s + pi/2))
    amp = 2 * abs(z) / n
    shift = ((-np.angle(z) - math.pi / 2) / k) % n
    assert shift == pytest.approx(U * t, rel=0.02)
    assert amp == pytest.approx(eps * math.exp(-nu * k * k * t), rel=0.02)


def test_uniform_flow_through_inlet_and_outflow_cells_is_a_fixed_point():
    nx, ny, nz = 12, 6, 5
    for faces, U in [((EQF, EQO, P, P, FS, FS), (0.06, 0.0, 0.0)), ((EQF, EQO, FS, FS, FS, FS), (0.06, 0.0, 0.0)),
                     ((EQF, EQO, EQF, EQF, FS, FS), (0.05, 0.03, 0.0))]:
        o = Oracle(nx, ny, nz, 1e-3, 0.1, 0.0, (0, 0, 0), faces)
        o.set_flags()
        o.set_inlet_profile(np.full(nz, U[0]), np.full(nz, U[1]), np.full(nz, U[2]))
        o.set_macros(None, np.full(o.shape, U[0]), np.full(o.shape, U[1]), np.full(o.shape, U[2]))
        G0 = o.get_state()
        o.step(40)
        assert np.abs(o.get_state() - G0).max() < 1e-15
        rho, ux, uy, uz = o.get_macros()
        assert np.abs(ux - U[0]).max() < 1e-15 and np.abs(uy - U[1]).max() < 1e-15 and np.abs(rho - 1).max() < 1e-14


def test_outflow_cell_copies_the_inward_neighbours_velocity_at_density_one():
    nx, ny, nz = 8, 4, 4
    rng = np.random.default_rng(9)
    o = Oracle(nx, ny, nz, 1e-2, 0.0, 0.0, (0, 0, 0), (EQF, EQO, P, P, FS, FS))
    o.set_flags()
    o.set_inlet_profile(np.full(nz, 0.03))
    o.set_macros(1 + 0.01 * rng.normal(size=o.shape), 0.03 + 0.01 * rng.normal(size=o.shape),
                 0.01 * rng.normal(size=o.shape), 0.01 * rng.normal(size=o.shape))
    for _ in range(3):
        before = o.get_macros()
        o.step(1)
        after = o.get_macros()
        assert np.abs(after[0][:, :, -1] - 1).max() < 1e-15
        for a in (1, 2, 3):
            np.testing.assert_allclose(after[a][:, :, -1], before[a][:, :, -2], atol=1e-15)
        # inlet cells never change
        np.testing.assert_allclose(after[1][:, :, 0], 0.03, atol=1e-16)
        assert np.abs(after[0][:, :, 0] - 1).max() < 1e-15


def test_local_macros_return_what_the_collision_used():
    """get_macros inverts the post-collision momentum m* = rho u + F_d/2: for k >= 1 it must return exactly the
    (rho,u) of step k's collision.  Checked through one cell: pull is the identity in a 1-cell periodic box."""
    rng = np.random.default_rng(4)
    nu0, Cs, fcor, F = 3e-3, 0.12, 0.03, (2e-5, -3e-5, 1e-5)
    o = Oracle(1, 1, 1, nu0, Cs, fcor, F, ALLP)
    o.set_flags()
    f = oracle.feq(1.02, np.array([0.04, -0.02, 0.03])) + 1e-4 * rng.normal(size=19)
    o.set_state(f.reshape(19, 1, 1, 1))
    o.step(1)
    _, rho_c, u_c, _ = oracle.collide_cell(f, nu0, Cs, fcor, F)
    rho, ux, uy, uz = o.get_macros()
    assert rho[0, 0, 0] == pytest.approx(rho_c, abs=1e-15)
    np.testing.assert_allclose([ux[0, 0, 0], uy[0, 0, 0], uz[0, 0, 0]], u_c, atol=1e-16)


def test_time_mean_accumulates_the_local_macros():
    nx, ny, nz = 6, 5, 4
    rng = np.random.default_rng(8)
    hm = np.zeros((ny, nx), dtype=np.int32)
    hm[1:3, 2:4] = 2
    o = Oracle(nx, ny, nz, 5e-3, 0.1, 1e-3, (1e-5, 0, 0), (P, P, P, P, WALL, FS))
    o.set_flags(hm)
    o.set_macros(None, 0.03 + 0.01 * rng.normal(size=o.shape), 0.01 * rng.normal(size=o.shape), None)
    o.mean_config(4, 3)
    acc = np.zeros((3,) + o.shape)
    cnt = 0
    for k in range(1, 15):
        o.step(1)
        if k >= 4 and (k - 4) % 3 == 0:
            m = o.get_macros()
            acc += np.stack(m[1:])
            cnt += 1
    mx, my, mz, n = o.get_mean()
    assert n == cnt == 4
    np.testing.assert_allclose(np.stack([mx, my, mz]), acc / cnt, atol=1e-16)
    assert np.all(mx[o.get_flags() == 1] == 0)


def test_outflow_cell_on_two_outflow_faces_uses_the_first_face_in_order():
    """DESIGN.md §4 reading 24 (outflow-edge owner): a cell on two EQ_OUTFLOW faces copies the velocity of its inward
    neighbour across the FIRST such face in the order x-, x+, y-, y+, z-, z+.  Faces (EQ_FIXED, EQ_OUTFLOW, FREE_SLIP,
    EQ_OUTFLOW, WALL, FREE_SLIP): the edge x = nx-1, y = ny-1 lies on x+ and y+; its neighbours across x+ and across y+
    hold different velocities, so the neighbour used is identified by brute force over all six candidates."""
    import oracle as O
    nx, ny, nz = 7, 6, 5
    faces = (3, 4, 2, 4, 1, 2)
    o = O.Oracle(nx, ny, nz, 1e-2, 0.0, 0.0, (0, 0, 0), faces)
    o.set_flags(None)
    rng = np.random.default_rng(5)
    o.set_inlet_profile(np.full(nz, 0.03))
    u0 = [0.02 + 0.01 * rng.random((nz, ny, nx)) for _ in range(3)]
    o.set_macros(None, *u0)
    cls = o.get_flags()
    assert cls[2, ny - 1, nx - 1] == 3 and cls[2, ny - 1, 3] == 3 and cls[2, 2, nx - 1] == 3
    before = o.get_macros()
    o.step(1)
    r, ux, uy, uz = o.get_macros()
    steps = {0: (1, 0, 0), 1: (-1, 0, 0), 2: (0, 1, 0), 3: (0, -1, 0), 4: (0, 0, 1), 5: (0, 0, -1)}  # x - n per face
    used = {}
    for z in range(nz):
        for (y, x) in [(ny - 1, nx - 1), (ny - 1, 3), (2, nx - 1)]:
            assert r[z, y, x] == pytest.approx(1.0, abs=1e-15)
            got = np.array([ux[z, y, x], uy[z, y, x], uz[z, y, x]])
            match = []
            for k, (dx, dy, dz) in steps.items():
                xs, ys, zs = x + dx, y + dy, z + dz
                if 0 <= xs < nx and 0 <= ys < ny and 0 <= zs < nz:
                    cand = np.array([before[1][zs, ys, xs], before[2][zs, ys, xs], before[3][zs, ys, xs]])
                    if np.abs(cand - got).max() < 1e-15:
                        match.append(k)
            assert len(match) == 1, (z, y, x, match)
            used[(y, x)] = match[0]
    assert used[(ny - 1, nx - 1)] == 1      # edge cell: x+ comes before y+
    assert used[(ny - 1, 3)] == 3           # y+ face proper
    assert used[(2, nx - 1)] == 1           # x+ face proper
    o.close()

"""Pins for the oracle's global flux-balancing correction (sign PAPER.md:185 "positive = outflow").

The correction is the least-squares-minimal change of the prescribed normal velocities that zeroes the net volume flux
through the open (EQ_FIXED) faces: a uniform shift along each cell's outward normal.  Pins: the invariant (net flux 0
afterwards), the closed form on a box whose imbalance is known by construction, minimality against other zero-flux
adjustments, tangential components untouched, idempotence, and the count of cells by brute force."""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def O(oracle_mod):
    return oracle_mod


def face_cells(nx, ny, nz, faces, flags):
    """Brute-force enumeration: (z, y, x, outward normal) of every EQ_FIXED cell, owner = first FIXED face it lies on."""
    out = []
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                if flags[z, y, x] != 2:
                    continue
                on = [x == 0, x == nx - 1, y == 0, y == ny - 1, z == 0, z == nz - 1]
                k = next(k for k in range(6) if on[k] and faces[k] == 3)
                n = np.zeros(3)
                n[k // 2] = 1.0 if k % 2 else -1.0
                out.append((z, y, x, n))
    return out


def make(O, faces, nx=10, ny=8, nz=6, seed=0):
    rng = np.random.default_rng(seed)
    o = O.Oracle(nx, ny, nz, 1e-2, 0.0, 0.0, (0, 0, 0), faces)
    hm = np.zeros((ny, nx), dtype=np.int32)
    hm[2:4, 0:2] = 3          # a building standing in the x- face: those face cells are SOLID, not open
    o.set_flags(hm)
    for k in range(6):
        if faces[k] == 3:
            axis = k // 2
            n1 = ny if axis == 0 else nx
            n2 = ny if axis == 2 else nz
            o.set_inlet_plane(k, 0.05 * rng.standard_normal((3, n2, n1)))
    o.set_macros()            # interior at rest (rho = 1, u = 0): the state is defined everywhere before it is compared
    return o


@pytest.mark.parametrize("faces", [(3, 3, 3, 3, 1, 3), (3, 4, 3, 3, 1, 2), (3, 3, 0, 0, 1, 2)])
def test_net_flux_vanishes_and_the_shift_is_uniform_along_the_normals(O, faces):
    nx, ny, nz = 10, 8, 6
    o = make(O, faces, nx, ny, nz)
    cells = face_cells(nx, ny, nz, faces, o.get_flags())
    r0, ux0, uy0, uz0 = [a.copy() for a in o.get_macros()]
    phi0 = sum(np.array([ux0[z, y, x], uy0[z, y, x], uz0[z, y, x]]) @ n for z, y, x, n in cells)
    before, after = o.balance_flux()
    assert before == pytest.approx(phi0, abs=1e-13)
    assert abs(after) < 1e-13
    r1, ux1, uy1, uz1 = o.get_macros()
    shift = phi0 / len(cells)
    for z, y, x, n in cells:
        du = np.array([ux1[z, y, x] - ux0[z, y, x], uy1[z, y, x] - uy0[z, y, x], uz1[z, y, x] - uz0[z, y, x]])
        assert np.abs(du + shift * n).max() < 1e-14          # same shift on every cell, along -n; tangential part untouched
        assert abs(r1[z, y, x] - 1.0) < 1e-14
    # every other cell is untouched
    mask = np.ones((nz, ny, nx), bool)
    for z, y, x, n in cells:
        mask[z, y, x] = False
    assert np.array_equal(ux1[mask], ux0[mask]) and np.array_equal(r1[mask], r0[mask])
    # idempotent
    b2, a2 = o.balance_flux()
    assert abs(b2) < 1e-13 and abs(a2) < 1e-13
    o.close()


def test_uniform_shift_is_the_minimal_adjustment(O):
    """Any other adjustment d with sum(d . n) = -Phi has a larger sum of squares (Cauchy-Schwarz); checked on random ones."""
    faces = (3, 3, 3, 3, 1, 3)
    nx, ny, nz = 10, 8, 6
    o = make(O, faces, nx, ny, nz, seed=5)
    cells = face_cells(nx, ny, nz, faces, o.get_flags())
    before, _ = o.balance_flux()
    N = len(cells)
    best = N * (before / N) ** 2
    rng = np.random.default_rng(6)
    for _ in range(50):
        d = rng.standard_normal(N)
        d += (-before - d.sum()) / N                   # project onto the constraint sum(d) = -Phi
        assert abs(d.sum() + before) < 1e-10
        assert (d ** 2).sum() >= best - 1e-15
    o.close()


def test_closed_form_on_a_box_with_a_known_imbalance(O):
    """Inflow U through all of x-, outflow V through all of x+ (no solids): Phi = (V - U) ny nz, shift = Phi / (2 ny nz)."""
    nx, ny, nz = 6, 5, 4
    U, V = 0.06, 0.02
    o = O.Oracle(nx, ny, nz, 1e-2, 0.0, 0.0, (0, 0, 0), (3, 3, 0, 0, 0, 0))
    o.set_flags(None)
    pl = np.zeros((3, nz, ny))
    pl[0] = U
    o.set_inlet_plane(0, pl)
    pl[0] = V
    o.set_inlet_plane(1, pl)
    before, after = o.balance_flux()
    assert before == pytest.approx((V - U) * ny * nz, rel=1e-12)      # negative: net inflow (PAPER.md:185 sign)
    r, ux, uy, uz = o.get_macros()
    assert np.allclose(ux[:, :, 0], 0.5 * (U + V), atol=1e-15) and np.allclose(ux[:, :, -1], 0.5 * (U + V), atol=1e-15)
    assert abs(after) < 1e-14
    o.close()

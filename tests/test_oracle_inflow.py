"""Pins for the synthetic inflow fluctuations of the oracle ("On-the-fly synthetic turbulent fluctuations are
superposed on this mean field"; Table 1 PAPER.md:86 "synthetic von Karman fluctuations on active inflow cells").

Reading (DESIGN.md §4 reading 21): u'(x,t) = 2 sum_n uhat_n cos(kappa_n.x + psi_n - omega_n t) sigma_n with
uhat_n = sqrt(E(|kappa_n|) dkappa_n), E = von Karman-Pao.  Nothing here re-types the spectrum or the mode sum; the pins
are what the mathematics fixes: the spectrum integrates to (3/2) u_rms^2, peaks at k/k_e = sqrt(12/5), rolls off as
k^(-5/3); one hand-placed mode gives a cosine of known zeros, sign pattern and time direction; time variance over a
full period is sum_n 2 uhat_n^2 sigma_n^2 (discrete orthogonality); omega = kappa.U_c makes the field a frozen pattern
carried by U_c; only cells whose mean velocity points inward carry u'; rho = 1; n = 0 restores the mean."""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def O(oracle_mod):
    return oracle_mod


def test_spectrum_integral_peak_and_inertial_slope(O):
    u_rms, k_e = 0.7, 0.3
    k = np.geomspace(1e-5, 1e10, 600001) * k_e                         # k^(-5/3) tail beyond: 1.5e-7 of the total
    E = O.vk_spectrum(k, u_rms, k_e)
    integral = np.sum(0.5 * (E[1:] + E[:-1]) * np.diff(k))
    assert integral == pytest.approx(1.5 * u_rms ** 2, rel=2.5e-4)    # alpha = 1.453 is the 4-digit rounding of 1.45276: +1.6e-4
    kk = np.linspace(1.0, 2.0, 200001) * k_e
    assert kk[np.argmax(O.vk_spectrum(kk, u_rms, k_e))] / k_e == pytest.approx(np.sqrt(12.0 / 5.0), abs=2e-5)
    hi = O.vk_spectrum(np.array([1e4, 2e4]) * k_e, u_rms, k_e)
    assert hi[1] / hi[0] == pytest.approx(2.0 ** (-5.0 / 3.0), rel=1e-6)
    lo = O.vk_spectrum(np.array([1e-4, 2e-4]) * k_e, u_rms, k_e)
    assert lo[1] / lo[0] == pytest.approx(16.0, rel=1e-6)             # k^4 at the large scales
    # energy scales with u_rms^2, shape only with k / k_e
    assert O.vk_spectrum([0.5], 2 * u_rms, k_e)[0] == pytest.approx(4 * O.vk_spectrum([0.5], u_rms, k_e)[0], rel=1e-14)
    assert O.vk_spectrum([1.0], u_rms, 2 * k_e)[0] * 2 * k_e == pytest.approx(O.vk_spectrum([0.5], u_rms, k_e)[0] * k_e, rel=1e-14)
    # Pao cut-off: the factor exp(-2 (k / k_eta)^2)
    assert O.vk_spectrum([0.9], u_rms, k_e, 1.8)[0] / O.vk_spectrum([0.9], u_rms, k_e)[0] == pytest.approx(np.exp(-0.5), rel=1e-14)


def box(O, faces=(3, 4, 0, 0, 1, 2), nx=8, ny=16, nz=8, U=0.05):
    o = O.Oracle(nx, ny, nz, 1e-2, 0.0, 0.0, (0, 0, 0), faces)
    o.set_flags(None)
    o.set_inlet_profile(np.full(nz, U))
    o.set_macros(None, np.full((nz, ny, nx), U), None, None)
    return o


def test_one_mode_is_a_cosine_with_the_stated_amplitude_zeros_and_time_direction(O):
    """kappa = (0, pi/4, 0), sigma = e_z, psi = 0: u'_z(y, t) = 2 uhat cos(pi y / 4 - omega t): peak at y = 0 (t = 0),
    zero at y = 2, trough at y = 4; with omega = pi/4 the crest moves to y = +1 after one step (phase -omega t)."""
    nx, ny, nz, U = 8, 16, 8, 0.05
    o = box(O)
    u_rms, k_e, dk = 0.01, 0.5, 0.125
    kap = np.pi / 4
    uhat = np.sqrt(O.vk_spectrum([kap], u_rms, k_e)[0] * dk)
    o.set_inflow_turbulence([[0, kap, 0, 0, 0, 1, 0.0, np.pi / 4, dk]], u_rms, k_e)
    r, ux, uy, uz = o.get_macros()
    w = uz[3, :, 0]
    assert w[0] == pytest.approx(2 * uhat, rel=1e-14) and w[4] == pytest.approx(-2 * uhat, rel=1e-14)
    assert abs(w[2]) < 1e-17 and abs(w[6]) < 1e-17 and w[1] == pytest.approx(2 * uhat * np.sqrt(0.5), rel=1e-13)
    assert np.abs(ux[:, :, 0] - U).max() < 1e-16 and np.abs(uy[:, :, 0]).max() < 1e-17   # sigma has no x, y part
    assert np.abs(r[:, :, 0] - 1).max() < 1e-15
    assert np.abs(uz[:, :, 0] - uz[3, :, 0][None, :]).max() < 1e-17                        # no z dependence
    o.step(1)
    w1 = o.get_macros()[3][3, :, 0]
    assert w1[1] == pytest.approx(2 * uhat, rel=1e-13)
    assert np.abs(w1 - np.roll(w, 1)).max() < 1e-15
    assert o.get_step() == 1
    o.close()


def test_time_variance_over_a_full_period_is_the_sum_of_mode_energies(O):
    """omega_n = 2 pi m_n / T with distinct integers m_n (m_n + m_k != 0 mod T): over T steps the modes are
    orthogonal, so mean_t u'_i = 0 and mean_t u'_i^2 = sum_n 2 uhat_n^2 sigma_n,i^2 exactly, at every cell."""
    from paper_2607_04516_b200 import workloads as W
    nx, ny, nz, U, T = 4, 6, 5, 0.05, 64
    o = box(O, nx=nx, ny=ny, nz=nz)
    modes = W.inflow_modes(6, 11, 0.1, 1.5)
    modes[:, 7] = 2 * np.pi * np.array([1, 2, 3, 5, 8, 13]) / T
    u_rms, k_e = 0.004, 0.4
    o.set_inflow_turbulence(modes, u_rms, k_e, 3.0)
    kmag = np.linalg.norm(modes[:, :3], axis=1)
    uhat2 = O.vk_spectrum(kmag, u_rms, k_e, 3.0) * modes[:, 8]
    want = (2 * uhat2[:, None] * modes[:, 3:6] ** 2).sum(axis=0)
    acc = np.zeros((3, nz, ny)); acc2 = np.zeros((3, nz, ny))
    for t in range(T):
        r, ux, uy, uz = o.get_macros()
        for a, f in enumerate((ux - U, uy, uz)):
            acc[a] += f[:, :, 0]; acc2[a] += f[:, :, 0] ** 2
        o.step(1)
    assert np.abs(acc / T).max() < 1e-16
    for a in range(3):
        assert np.abs(acc2[a] / T - want[a]).max() < 1e-15 * max(1.0, want[a] / 1e-6) and want[a] > 1e-8
    o.close()


def test_frozen_pattern_is_carried_by_the_convection_velocity(O):
    """omega = kappa . U_c  =>  u'(x, t) = u'(x - U_c t, 0).  U_c = (0, 1, 0): one cell per step in +y."""
    from paper_2607_04516_b200 import workloads as W
    o = box(O, ny=24)
    modes = W.inflow_modes(12, 5, 0.1, 2.0, convect=(0.0, 1.0, 0.0))
    o.set_inflow_turbulence(modes, 0.005, 0.5)
    f0 = [a[:, :, 0].copy() for a in o.get_macros()[1:]]
    o.step(3)
    f3 = [a[:, :, 0] for a in o.get_macros()[1:]]
    for a, b in zip(f0, f3):
        assert np.abs(b[:, 3:] - a[:, :-3]).max() < 1e-15
        assert np.abs(b - a).max() > 1e-4          # the pattern did move
    o.close()


def test_only_active_inflow_cells_fluctuate_and_switching_off_restores_the_mean(O):
    """Four EQ_FIXED lateral faces under a mean wind (U, V, 0) with U, V > 0: x- and y- cells see inflow (ub.n < 0),
    x+ and y+ cells outflow: they keep the mean.  Tangential-only faces (z+ here, w = 0) are not 'inflow' either."""
    from paper_2607_04516_b200 import workloads as W
    nx, ny, nz, U, V = 10, 9, 6, 0.05, 0.02
    o = O.Oracle(nx, ny, nz, 1e-2, 0.0, 0.0, (0, 0, 0), (3, 3, 3, 3, 1, 3))
    o.set_flags(None)
    o.set_inlet_profile(np.full(nz, U), np.full(nz, V))
    o.set_macros(None, np.full((nz, ny, nx), U), np.full((nz, ny, nx), V), None)
    m0 = [a.copy() for a in o.get_macros()]
    o.set_inflow_turbulence(W.inflow_modes(10, 3, 0.2, 2.0), 0.005, 0.5)
    o.step(2)
    r, ux, uy, uz = o.get_macros()
    d = np.sqrt((ux - U) ** 2 + (uy - V) ** 2 + uz ** 2)
    fl = o.get_flags()
    assert (fl[:, :, 0] == 2).all() and (fl[nz - 1] == 2).all()
    # x- face (owner face 0 also on its edges with y and z faces): active
    assert d[:, :, 0].min() > 1e-5
    # y- face away from x = 0 (owner face 2): active; x+ (owner 1) and y+ away from x = 0 (owner 3): mean kept
    assert d[:nz - 1, 0, 1:nx - 1].min() > 1e-5
    assert d[:, :, nx - 1].max() < 1e-16
    assert d[:nz - 1, ny - 1, 1:nx - 1].max() < 1e-16
    # top face interior (owner 5, w_mean = 0: not inflow): mean kept
    assert d[nz - 1, 1:ny - 1, 1:nx - 1].max() < 1e-16
    assert np.abs(r[fl == 2] - 1).max() < 1e-15
    # the mean cannot be replaced while fluctuations ride on it
    with pytest.raises(RuntimeError):
        o.set_inlet_profile(np.full(nz, U))
    with pytest.raises(RuntimeError):
        o.balance_flux()
    o.set_inflow_turbulence(None)
    m1 = o.get_macros()
    for a, b in zip(m0, m1):
        assert np.abs(a[fl == 2] - b[fl == 2]).max() < 1e-16
    o.set_inlet_profile(np.full(nz, U), np.full(nz, V))   # allowed again
    o.close()


def test_fluctuations_enter_the_flow_and_mass_flux_stays_bounded(O):
    """The fluid behind an active inlet picks the fluctuations up (downstream cells deviate from the uniform fixed point
    the same box keeps without them), and the state stays finite and near rho = 1."""
    from paper_2607_04516_b200 import workloads as W
    o = box(O, faces=(3, 4, 0, 0, 2, 2), nx=24, ny=12, nz=8)
    o.step(20)
    assert np.abs(o.get_macros()[3]).max() < 1e-14           # fixed point without fluctuations (rounding only)
    o.set_inflow_turbulence(W.inflow_modes(16, 9, 0.2, 2.0, convect=(0.05, 0, 0)), 0.004, 0.5)
    o.step(60)
    r, ux, uy, uz = o.get_macros()
    assert np.isfinite(ux).all() and np.abs(r - 1).max() < 0.05
    assert np.abs(uz[:, :, 3]).max() > 1e-4 and np.abs(uy[:, :, 3]).max() > 1e-4
    o.close()


def test_active_inflow_threshold_is_1e7_strict_and_in_lattice_units(O):
    """DESIGN.md §4 reading 21: a cell is an 'active inflow cell' iff ub.n < -1e-7 (n outward, lattice units).  One x-
    face whose cells carry different mean normal components straddling the constant: +5e-8 and +9.9e-8 (inward by less
    than the threshold) and exactly 1e-7 (strict '<') keep the mean EXACTLY; 1.01e-7 and 2e-7 fluctuate.  The same
    magnitudes with the opposite sign (outflow through x-) never fluctuate.  A typo in the constant (1e-6, 1e-8), a
    '<=' or a dropped sign fails here."""
    from paper_2607_04516_b200 import workloads as W
    nx, ny, nz = 6, 10, 4
    o = O.Oracle(nx, ny, nz, 1e-2, 0.0, 0.0, (0, 0, 0), (3, 4, 0, 0, 2, 2))
    o.set_flags(None)
    un = np.array([5e-8, 9.9e-8, 1e-7, 1.01e-7, 2e-7, -5e-8, -1e-7, -1.01e-7, -2e-7, 1e-6])   # u_x per y; x- face: ub.n = -u_x
    plane = np.zeros((3, nz, ny))
    plane[0] = un[None, :]
    plane[1] = 0.01                                     # a tangential part: must not enter the test
    o.set_inlet_plane(0, plane)
    o.set_macros()
    o.set_inflow_turbulence(W.inflow_modes(8, 21, 0.2, 2.0), 0.01, 0.5)
    active = np.array([False, False, False, True, True, False, False, False, False, True])
    for _ in range(3):
        r, ux, uy, uz = o.get_macros()
        dev = np.sqrt((ux[:, :, 0] - un[None, :]) ** 2 + (uy[:, :, 0] - 0.01) ** 2 + uz[:, :, 0] ** 2)
        assert dev[:, ~active].max() < 1e-15, "a cell below the threshold must keep its mean (up to the rounding of the moment sums)"
        assert dev[:, active].min() > 1e-4, "a cell above the threshold must fluctuate"
        o.step(1)
    o.close()

"""Parity of the fused flow + thermal step (lbm_set_thermal / lbm_set_theta / lbm_get_theta; SURVEY.md §8(f) rank 3,
PAPER.md:89, :121; DESIGN.md §4 reading 23) against the CPU FP64 oracle through the C ABI.
Bars: max-abs(rho, u, theta - theta_ref) <= 1e-5 after 100 steps (FP32), <= 2e-12 (FP64 instantiation)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL32 = 1e-5
TOL64 = 2e-12
P, W, FS = 0, 1, 2


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2607_04516_b200 import binding, build
    build.build()
    return binding


def pair(B, nx, ny, nz, faces, hm, nu0, Cs, fcor, F, alpha, gb, tref, theta, u0=None, fp64=False, want_mean=False, inplace=False):
    from oracle import Oracle
    o = Oracle(nx, ny, nz, nu0, Cs, fcor, F, faces)
    o.set_flags(hm)
    sim = B.Lbm(nx, ny, nz, nu0, Cs, fcor, F, faces, fp64=fp64, want_mean=want_mean, inplace=inplace)
    sim.set_flags(hm)
    np.testing.assert_array_equal(sim.get_flags(), o.get_flags())
    u0 = u0 or (None, None, None)
    o.set_macros(None, *u0)
    sim.set_macros(None, *u0, f64=True)
    o.set_thermal(alpha, gb, tref)
    sim.set_thermal(alpha, gb, tref)
    o.set_theta(theta, *u0)
    sim.set_theta(theta, *u0, f64=True)
    return sim, o


def errs(sim, o, tref):
    g = [a.cpu().numpy().astype(np.float64) for a in sim.get_macros(f64=True)]
    r = o.get_macros()
    e_flow = max(float(np.abs(a - b).max()) for a, b in zip(g, r))
    th = sim.get_theta(f64=True).cpu().numpy()
    assert np.isfinite(th).all()
    e_th = float(np.abs(th - o.get_theta()).max())
    # and the seven thermal populations themselves (lbm_get_thermal_state against the oracle's), boundary cells included: their
    # first moment is the heat flux, which theta alone does not see
    e_th = max(e_th, float(np.abs(sim.get_thermal_state() - o.get_thermal_state()).max()))
    return e_flow, e_th


FACES = [(P, P, P, P, P, P), (W, FS, P, P, W, FS), (FS, FS, FS, FS, FS, FS), (W, W, W, W, W, W), (FS, W, P, P, FS, W)]


@pytest.mark.parametrize("inplace", [False, True])    # the flow lattice on one buffer; the thermal one stays double
@pytest.mark.parametrize("fp64", [False, True])
@pytest.mark.parametrize("faces", FACES)
def test_thermal_parity_ragged_boxes_with_solids(B, faces, fp64, inplace):
    rng = np.random.default_rng(11 + FACES.index(faces))
    for nx, ny, nz in [(33, 7, 9), (70, 5, 12)]:
        hm = np.zeros((ny, nx), np.int32)
        hm[1:4, 5:11] = 4
        hm[ny - 2, nx - 9:nx - 3] = 2
        theta = 1.0 + 0.3 * rng.standard_normal((nz, ny, nx))
        u0 = tuple(0.02 * rng.standard_normal((nz, ny, nx)) for _ in range(3))
        sim, o = pair(B, nx, ny, nz, faces, hm, 2e-3, 0.1, 1e-3, (1e-6, 0, 0), 0.01, 2e-3, 1.0, theta, u0, fp64=fp64, inplace=inplace)
        sim.step(101); o.step(101)
        e_flow, e_th = errs(sim, o, 1.0)
        tol = TOL64 if fp64 else TOL32
        assert e_flow <= tol and e_th <= tol, (faces, (nx, ny, nz), e_flow, e_th)
        sim.close(); o.close()


@pytest.mark.parametrize("fp64", [False, True])
def test_density_current_parity_and_time_mean(B, fp64):
    from paper_2607_04516_b200 import workloads as Wl
    nx, ny, nz = 128, 2, 32
    faces, theta = Wl.density_current(nx, nz, ny, d_theta=-15.0, theta_ref=300.0)
    hm = np.zeros((ny, nx), np.int32)
    sim, o = pair(B, nx, ny, nz, faces, hm, 1e-3, 0.1, 0.0, (0, 0, 0), 1e-3, 2e-5, 300.0, theta, fp64=fp64, want_mean=True)
    sim.mean_config(50, 10); o.mean_config(50, 10)
    sim.step(200); o.step(200)
    e_flow, e_th = errs(sim, o, 300.0)
    tol = TOL64 if fp64 else TOL32
    # theta' spans 15 K: the thermal bar is relative to that span (FP32 storage is shifted by theta_ref)
    assert e_flow <= tol and e_th <= 15.0 * tol, (e_flow, e_th)
    gm = sim.get_mean(f64=True); om = o.get_mean()
    assert gm[3] == om[3] == 16
    assert max(float(np.abs(a.cpu().numpy() - b).max()) for a, b in zip(gm[:3], om[:3])) <= tol
    # the cold pool sinks: downward motion under the blob's centre
    uz = o.get_macros()[3]
    assert uz[nz // 2, 0, nx // 2] < -1e-4
    sim.close(); o.close()


def test_heat_and_mass_conserved_on_the_gpu_fp64(B):
    nx, ny, nz = 40, 6, 20
    rng = np.random.default_rng(5)
    hm = np.zeros((ny, nx), np.int32); hm[2:4, 10:18] = 7
    theta = 2.0 + 0.5 * rng.standard_normal((nz, ny, nx))
    sim, o = pair(B, nx, ny, nz, (W, FS, P, P, W, FS), hm, 5e-3, 0.1, 1e-3, (0, 0, 0), 0.02, 1e-3, 2.0, theta, fp64=True)
    fluid = sim.get_flags() == 0
    s0 = sim.get_theta(f64=True).cpu().numpy()[fluid].sum()
    sim.step(300)
    s1 = sim.get_theta(f64=True).cpu().numpy()[fluid].sum()
    assert abs(s1 - s0) <= 1e-12 * abs(s0)
    rho = sim.get_macros(f64=True)[0].cpu().numpy()
    assert abs(rho[fluid].sum() - fluid.sum()) <= 1e-11 * fluid.sum()
    sim.close(); o.close()


def test_zero_buoyancy_leaves_the_flow_unchanged(B):
    # g_beta = 0: the fused kernel's flow half is the plain step's arithmetic; the two instantiations may contract
    # multiply-adds differently around the (now per-cell) F_z, so equal up to FP32 rounding order, not bit for bit
    nx, ny, nz = 48, 9, 10
    rng = np.random.default_rng(6)
    hm = np.zeros((ny, nx), np.int32); hm[3:6, 12:20] = 5
    u0 = tuple(0.02 * rng.standard_normal((nz, ny, nx)) for _ in range(3))
    faces = (P, P, FS, FS, W, FS)
    a = B.Lbm(nx, ny, nz, 2e-3, 0.1, 1e-3, (1e-6, 0, 0), faces, want_mean=False)
    b = B.Lbm(nx, ny, nz, 2e-3, 0.1, 1e-3, (1e-6, 0, 0), faces, want_mean=False)
    for s in (a, b):
        s.set_flags(hm); s.set_macros(None, *u0, f64=True)
    b.set_thermal(0.01, 0.0, 1.0)
    b.set_theta(1.0 + 0.1 * rng.standard_normal((nz, ny, nx)), f64=True)
    a.step(37); b.step(37)
    assert float(np.abs(a.get_state(out="host") - b.get_state(out="host")).max()) <= 1e-7
    a.close(); b.close()


def test_thermal_error_behaviour(B):
    sim = B.Lbm(8, 8, 8, 1e-2)  # default faces carry EQ_FIXED / EQ_OUTFLOW
    sim.set_flags(np.zeros((8, 8), np.int32))
    with pytest.raises(B.LbmError):
        sim.get_theta()
    with pytest.raises(B.LbmError):
        sim.set_inlet_theta(np.ones(8, np.float32))     # thermal lattice off
    sim.set_boundaries([P] * 6)
    with pytest.raises(B.LbmError):
        sim.set_thermal(0.0, 0.0, 1.0)  # alpha must be > 0
    sim.set_thermal(0.01, 1e-3, 1.0)
    with pytest.raises(B.LbmError):
        sim.set_theta()  # flags were invalidated by set_boundaries
    sim.set_flags(np.zeros((8, 8), np.int32))

    sim.set_macros(); sim.set_theta()
    sim.step(3)
    assert float(np.abs(sim.get_theta().cpu().numpy() - 1.0).max()) == 0.0  # isothermal rest state is exact
    sim.close()


def test_thermal_full_size_city_box_parity_and_conservation(B):
    """The launch configuration `bench.py --workload thermal` times: closed 400x400x100 city box (config 3's heightmap),
    theta = 300 + N(0,1) K, buoyancy on.  Whole-field parity against the oracle after 30 steps, and heat conservation."""
    from paper_2607_04516_b200 import workloads as Wl
    from oracle import Oracle
    wl = Wl.thermal_city()
    alpha, gb, tref = wl.extra["thermal"]
    theta = wl.extra["theta"]
    sim = B.from_workload(wl, want_mean=False)
    o = Oracle(wl.nx, wl.ny, wl.nz, wl.nu0, wl.Cs, wl.f_cor, wl.F, wl.faces)
    o.set_flags(wl.height)
    o.set_macros()
    o.set_thermal(alpha, gb, tref)
    o.set_theta(theta.astype(np.float64))
    fluid = sim.get_flags() == 0
    np.testing.assert_array_equal(sim.get_flags(), o.get_flags())
    s0 = float((sim.get_theta(f64=True).cpu().numpy() - tref)[fluid].sum())
    sim.step(30); o.step(30)
    e_flow, e_th = errs(sim, o, tref)
    assert e_flow <= TOL32 and e_th <= TOL32, (e_flow, e_th)
    th = sim.get_theta(f64=True).cpu().numpy() - tref
    # sum of theta' over 1.56e7 fluid cells of O(1) K each: FP32 rounding of the stored populations only
    assert abs(float(th[fluid].sum()) - s0) <= 1e-6 * float(np.abs(th[fluid]).sum())
    sim.close(); o.close()


@pytest.mark.parametrize("faces", [(P, P, P, P, P, P), (W, FS, P, P, W, FS), (FS, FS, W, W, FS, FS)])
def test_thermal_parity_degenerate_boxes(B, faces):
    # boxes one cell thick along one or two axes (every pull wraps / reflects / bounces onto the cell itself)
    rng = np.random.default_rng(21)
    for nx, ny, nz in [(1, 1, 3), (5, 1, 1), (1, 4, 1), (6, 5, 4), (32, 1, 2)]:
        hm = np.zeros((ny, nx), np.int32)
        if nx >= 5 and nz >= 2:
            hm[0, 2] = 1
        theta = 1.0 + 0.3 * rng.standard_normal((nz, ny, nx))
        u0 = tuple(0.02 * rng.standard_normal((nz, ny, nx)) for _ in range(3))
        sim, o = pair(B, nx, ny, nz, faces, hm, 2e-3, 0.1, 1e-3, (1e-6, 0, 0), 0.01, 2e-3, 1.0, theta, u0, fp64=True)
        sim.step(40); o.step(40)
        e_flow, e_th = errs(sim, o, 1.0)
        assert e_flow <= TOL64 and e_th <= TOL64, (faces, (nx, ny, nz), e_flow, e_th)
        sim.close(); o.close()


def _paper_fronts():
    import os
    rows = [l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "density_current_fronts.txt"))
            if l.strip() and not l.startswith("#")]
    return [(int(r[0]), float(r[1]), float(r[2])) for r in rows]


def _gpu_fronts(B, dx):
    from paper_2607_04516_b200 import workloads as Wl
    b = Wl.density_current_benchmark(dx, 0.1)
    sim = B.Lbm(b["nx"], b["ny"], b["nz"], b["nu"], 0.0, 0.0, (0, 0, 0), b["faces"], want_mean=False)
    sim.set_flags(np.zeros((b["ny"], b["nx"]), np.int32))
    sim.set_macros()
    sim.set_thermal(b["alpha"], b["g_beta"], b["theta_ref"])
    sim.set_theta(b["theta"], f64=True)
    got = {}
    for T, _, _ in _paper_fronts():
        sim.step(int(round(T / b["dt"])) - sim.get_step())
        got[T] = Wl.front_position_km(sim.get_theta(f64=True).cpu().numpy()[:, 0, :], b["x_m"])
    sim.close()
    return b, got


def test_density_current_fronts_gpu_vs_oracle_at_100m(B):
    """The benchmark of PAPER.md:121-125 through the C ABI in FP32, 3150 steps: front positions equal the oracle's to 0.5 %
    (a laminar AV75 run: no chaotic divergence) and the paper's printed ones within 8 %."""
    from oracle import Oracle
    from paper_2607_04516_b200 import workloads as Wl
    b, got = _gpu_fronts(B, 100.0)
    o = Oracle(b["nx"], b["ny"], b["nz"], b["nu"], 0.0, 0.0, (0, 0, 0), b["faces"])
    o.set_flags(); o.set_macros(); o.set_thermal(b["alpha"], b["g_beta"], b["theta_ref"]); o.set_theta(b["theta"])
    for T, ref, plat in _paper_fronts():
        o.step(int(round(T / b["dt"])) - o.get_step())
        xo = Wl.front_position_km(o.get_theta()[:, 0, :], b["x_m"])
        assert abs(got[T] / xo - 1.0) < 5e-3, (T, got[T], xo)
        assert abs(got[T] / ref - 1.0) < 0.08 and abs(got[T] / plat - 1.0) < 0.08, (T, got[T], ref, plat)
    o.close()


def test_density_current_fronts_gpu_at_25m_against_the_papers_printed_values(B):
    """The paper's coarser comparison grid (25 m): 1024 x 256 cells, 12 600 steps on the GPU path."""
    b, got = _gpu_fronts(B, 25.0)
    for T, ref, plat in _paper_fronts():
        assert abs(got[T] / ref - 1.0) < 0.08 and abs(got[T] / plat - 1.0) < 0.08, (T, got[T], ref, plat)
    print("density current 25 m fronts (km):", got)


@pytest.mark.parametrize("fp64", [False, True])
def test_thermal_checkpoint_restarts_exactly(B, fp64):
    """lbm_get_state + lbm_get_thermal_state + the step counter are a complete checkpoint of a thermal run: a fresh handle
    loaded with them continues like the uninterrupted one (mailboxes and ghost slots of both lattices are rebuilt by the
    set calls) — bit for bit on the FP32 handle; on the FP64 handle up to the last bit, because the checkpoint holds the
    unshifted populations and (g + w) - w is not g in the handle's own precision."""
    nx, ny, nz = 36, 10, 14
    rng = np.random.default_rng(8)
    hm = np.zeros((ny, nx), np.int32); hm[3:6, 8:14] = 5
    theta = 1.0 + 0.2 * rng.standard_normal((nz, ny, nx))
    args = (nx, ny, nz, 2e-3, 0.1, 1e-3, (1e-6, 0, 0), (P, P, FS, W, W, FS))

    def fresh():
        s = B.Lbm(*args, fp64=fp64)
        s.set_flags(hm)
        s.set_macros()
        s.set_thermal(0.01, 2e-3, 1.0)
        return s
    a = fresh()
    a.set_theta(theta, f64=True)
    a.step(40)
    f, hpop, k = a.get_state(out="host"), a.get_thermal_state(), a.get_step()
    assert hpop.shape == (7, nz, ny, nx)
    th = a.get_theta(out="host", f64=True)
    np.testing.assert_allclose(hpop.sum(axis=0)[hm[None] <= np.arange(nz)[:, None, None]], th[hm[None] <= np.arange(nz)[:, None, None]], rtol=0, atol=1e-6 if not fp64 else 1e-13)
    b = fresh()
    b.set_state(f); b.set_thermal_state(hpop); b.set_step(k)
    a.step(25); b.step(25)
    if fp64:
        np.testing.assert_allclose(a.get_state(out="host"), b.get_state(out="host"), rtol=0, atol=1e-14)
        np.testing.assert_allclose(a.get_thermal_state(), b.get_thermal_state(), rtol=0, atol=1e-14)
    else:
        np.testing.assert_array_equal(a.get_state(out="host"), b.get_state(out="host"))
        np.testing.assert_array_equal(a.get_thermal_state(), b.get_thermal_state())
    assert a.get_step() == b.get_step() == 65
    a.close(); b.close()


# ---- fixed-temperature walls (DESIGN.md §4 reading 26) -------------------------------------------------------------------

def walls_pair(B, nx, ny, nz, faces, hm, nu0, alpha, gb, tref, on, tw, theta, fp64, Cs=0.1, fcor=0.0, F=(0, 0, 0)):
    """like pair(), with the held walls set BEFORE the thermal state is written (the mailboxes then carry the wall rule)"""
    from oracle import Oracle
    o = Oracle(nx, ny, nz, nu0, Cs, fcor, F, faces)
    o.set_flags(hm)
    sim = B.Lbm(nx, ny, nz, nu0, Cs, fcor, F, faces, fp64=fp64)
    sim.set_flags(hm)
    o.set_macros(); sim.set_macros()
    o.set_thermal(alpha, gb, tref); sim.set_thermal(alpha, gb, tref)
    o.set_thermal_walls(on, tw); sim.set_thermal_walls(on, tw)
    o.set_theta(theta); sim.set_theta(theta, f64=True)
    return sim, o


@pytest.mark.parametrize("fp64", [False, True])
def test_held_walls_parity_with_buildings_and_mixed_faces(B, fp64):
    """Heated ground (held), adiabatic lid (WALL, not held), a held side wall, periodic y, buildings standing on the heated
    ground (their surfaces stay adiabatic), buoyancy, LES, Coriolis: 100 steps against the oracle."""
    nx, ny, nz = 44, 9, 16
    rng = np.random.default_rng(21)
    hm = np.zeros((ny, nx), np.int32); hm[2:6, 10:17] = 6; hm[5:8, 28:33] = 3
    theta = 1.0 + 0.05 * rng.standard_normal((nz, ny, nx))
    on, tw = [1, 0, 0, 0, 1, 0], [0.7, 0, 0, 0, 1.6, 0]
    sim, o = walls_pair(B, nx, ny, nz, (W, W, P, P, W, W), hm, 4e-3, 0.02, 3e-3, 1.0, on, tw, theta, fp64, fcor=1e-3)
    sim.step(100); o.step(100)
    e_flow, e_th = errs(sim, o, 1.0)
    tol = TOL64 if fp64 else TOL32
    assert e_flow <= tol and e_th <= tol, (e_flow, e_th)
    th = o.get_theta()
    assert th[0][hm == 0].mean() > 1.2          # the ground does heat the air above it
    sim.close(); o.close()


def test_conduction_profile_and_rayleigh_benard_box_on_the_gpu(B):
    """The two closed-form set-ups of tests/test_oracle_thermal.py on the CUDA path: (i) pure conduction between held
    plates converges to the exact linear profile on the FP64 kernels (1e-10) and the FP32 kernels (1e-5); (ii) the
    Rayleigh-Benard box at 1.1 Ra_c: FP64 kernels follow the oracle's growing roll for 4000 steps to rounding order
    relative to its amplitude."""
    from oracle import Oracle
    nz = 10
    zeta = np.arange(nz) + 0.5
    exact = 1.0 + (0.25 - 1.0) * zeta / nz
    for fp64, tol in ((True, 1e-10), (False, 1e-5)):
        sim = B.Lbm(4, 3, nz, 0.05, 0.0, 0.0, (0, 0, 0), (P, P, P, P, W, W), fp64=fp64)
        sim.set_flags(None); sim.set_macros()
        sim.set_thermal(0.12, 0.0, 0.6)
        sim.set_thermal_walls([0, 0, 0, 0, 1, 1], [0, 0, 0, 0, 1.0, 0.25])
        sim.set_theta(np.full((nz, 3, 4), 0.6), f64=True)
        sim.step(6000)
        th = sim.get_theta(out="host", f64=True)
        assert np.abs(th - exact[:, None, None]).max() < tol, fp64
        sim.close()
    H, nu, alpha, Ra = 16, 0.05, 0.05, 1.1 * 1707.76
    nx = 2 * H
    gb = Ra * nu * alpha / H ** 3
    z = (np.arange(H) + 0.5) / H
    mode = np.sin(np.pi * z)[:, None] * np.cos(2 * np.pi * (np.arange(nx) + 0.5) / nx)[None, :]
    theta = ((1.0 - z)[:, None] + 1e-4 * mode)[:, None, :]
    sim, o = walls_pair(B, nx, 1, H, (P, P, P, P, W, W), None, nu, alpha, gb, 0.5, [0, 0, 0, 0, 1, 1], [0, 0, 0, 0, 1.0, 0.0],
                        theta, True, Cs=0.0)
    a0 = None
    for _ in range(4):
        sim.step(1000); o.step(1000)
        wo = o.get_macros()[3]
        wg = sim.get_macros(f64=True)[3].cpu().numpy()
        amp = np.abs(wo).max()
        assert np.abs(wg - wo).max() <= 1e-9 * amp + 1e-15
        a0 = a0 or amp
    assert amp > 1.1 * a0                        # supercritical: the roll grows
    sim.close(); o.close()


def test_thermal_walls_argument_errors(B):
    sim = B.Lbm(8, 8, 8, 1e-2, 0.0, 0.0, (0, 0, 0), (P, P, FS, FS, W, W))
    sim.set_flags(None)
    with pytest.raises(B.LbmError):
        sim.set_thermal_walls([0, 0, 0, 0, 1, 1], [0] * 6)          # thermal lattice off
    sim.set_thermal(0.01, 0.0, 0.0)
    with pytest.raises(B.LbmError):
        sim.set_thermal_walls([0, 0, 1, 0, 0, 0], [0] * 6)          # a FREE_SLIP face cannot be held
    with pytest.raises(B.LbmError):
        sim.set_thermal_walls([0, 0, 0, 0, 1, 0], [0, 0, 0, 0, float("nan"), 0])
    sim.set_thermal_walls([0, 0, 0, 0, 1, 1], [9, 9, 9, 9, 1.0, 0.0])   # entries of faces not held are ignored
    sim.close()


# ---- thermal lattice on open faces (DESIGN.md §4 reading 27) ---------------------------------------------------------------

EQF, EQO = 3, 4


def open_pair(B, nx, ny, nz, faces, hm, fp64, gb=3e-4, alpha=0.02, tref=1.0, seed=0, want_mean=False, inplace=False):
    from oracle import Oracle
    rng = np.random.default_rng(seed)
    prof = (0.05 * np.log((np.arange(nz) + 0.5) / 0.1) / np.log(nz / 0.1)).clip(0)
    thb = tref + 0.4 * np.exp(-np.arange(nz) / 4.0)            # warm air near the ground at the inlet
    u0 = np.broadcast_to(prof[:, None, None], (nz, ny, nx)).copy()
    th0 = tref + 0.05 * rng.standard_normal((nz, ny, nx))
    args = (nx, ny, nz, 3e-3, 0.1, 1e-3, (1e-6, 0, 0), faces)
    o = Oracle(*args)
    sim = B.Lbm(*args, fp64=fp64, want_mean=want_mean, inplace=inplace)
    for obj, kw in ((o, {}), (sim, {"f64": True})):
        obj.set_flags(hm)
        obj.set_inlet_profile(prof, 0.1 * prof, None, **kw)
        obj.set_macros(None, u0, None, None, **kw)
        obj.set_thermal(alpha, gb, tref)
        obj.set_inlet_theta(thb, **kw)
        obj.set_theta(th0, u0, None, None, **kw)
    return sim, o, prof, thb


@pytest.mark.parametrize("inplace", [False, True])
@pytest.mark.parametrize("fp64", [False, True])
@pytest.mark.parametrize("faces", [(EQF, EQO, P, P, W, FS), (EQF, EQO, FS, FS, W, FS), (EQF, EQO, EQF, EQF, W, FS), (EQO, EQF, W, FS, P, P)])
def test_open_faces_parity(B, faces, fp64, inplace):
    """Inlet with a prescribed theta_b(z) and u_b(z), outflow copying theta and u, buildings, buoyancy, LES, Coriolis, a body
    force: rho, u, theta against the oracle after 100 steps; the state right after set-up too (boundary cells included)."""
    nx, ny, nz = 52, 14, 12
    hm = np.zeros((ny, nx), np.int32); hm[3:8, 14:20] = 5; hm[8:12, 30:36] = 3
    sim, o, prof, thb = open_pair(B, nx, ny, nz, faces, hm, fp64, seed=FACES.index(FACES[0]) + len(faces), inplace=inplace)
    tol = TOL64 if fp64 else TOL32
    e_flow, e_th = errs(sim, o, 1.0)
    assert e_flow <= tol and e_th <= tol, ("set-up", faces, e_flow, e_th)
    sim.step(100); o.step(100)
    e_flow, e_th = errs(sim, o, 1.0)
    assert e_flow <= tol and e_th <= tol, (faces, e_flow, e_th)
    th = o.get_theta()
    assert np.abs(th - 1.0).max() > 0.05                         # the warm inflow is really there
    sim.close(); o.close()


def test_open_faces_boundary_updates_mean_and_checkpoint(B):
    """A new velocity profile keeps theta_b and refreshes the inlet cells; the fused time mean runs on EQ cells too; state +
    thermal state + step restart a run with open faces exactly (FP32)."""
    nx, ny, nz = 40, 8, 10
    hm = np.zeros((ny, nx), np.int32); hm[2:5, 12:17] = 4
    faces = (EQF, EQO, P, P, W, FS)
    sim, o, prof, thb = open_pair(B, nx, ny, nz, faces, hm, False, seed=5, want_mean=True)
    sim.step(20); o.step(20)
    for obj, kw in ((o, {}), (sim, {"f64": True})):
        obj.set_inlet_profile(1.2 * prof, None, None, **kw)
        obj.mean_config(25, 5)
    e_flow, e_th = errs(sim, o, 1.0)
    assert e_flow <= TOL32 and e_th <= TOL32
    sim.step(40); o.step(40)
    e_flow, e_th = errs(sim, o, 1.0)
    assert e_flow <= TOL32 and e_th <= TOL32, (e_flow, e_th)
    gm = sim.get_mean(f64=True); om = o.get_mean()
    assert gm[3] == om[3] == 8
    assert max(float(np.abs(a.cpu().numpy() - b).max()) for a, b in zip(gm[:3], om[:3])) <= TOL32
    # checkpoint
    f, hpop, k = sim.get_state(out="host"), sim.get_thermal_state(), sim.get_step()
    b = B.Lbm(nx, ny, nz, 3e-3, 0.1, 1e-3, (1e-6, 0, 0), faces)
    b.set_flags(hm)
    b.set_inlet_profile(1.2 * prof, None, None, f64=True)
    b.set_macros()
    b.set_thermal(0.02, 3e-4, 1.0)
    b.set_inlet_theta(thb, f64=True)
    b.set_state(f); b.set_inlet_profile(1.2 * prof, None, None, f64=True); b.set_thermal_state(hpop); b.set_step(k)
    sim.step(15); b.step(15)
    ga = [a.cpu().numpy() for a in sim.get_macros()] + [sim.get_theta(out="host")]
    gb_ = [a.cpu().numpy() for a in b.get_macros()] + [b.get_theta(out="host")]
    assert max(float(np.abs(x - y).max()) for x, y in zip(ga, gb_)) <= 2e-6
    sim.close(); o.close(); b.close()


@pytest.mark.parametrize("inplace", [False, True])
@pytest.mark.parametrize("fp64", [False, True])
@pytest.mark.parametrize("faces", [(EQF, EQO, EQF, EQF, W, EQF), (EQF, EQO, P, P, W, FS), (P, P, P, P, W, FS)])
def test_damping_zones_together_with_the_thermal_lattice(B, faces, fp64, inplace):
    """The paper's open-boundary damping (top sponge + lateral buffer nudging) on a thermal run: the relaxation
    acceleration and the buoyancy share one implicit half-force solve (oracle pin: test_oracle_thermal.py
    ::test_buoyancy_against_a_uniform_damping_zone_settles_at_a_over_sigma).  Buildings, warm inflow, LES, Coriolis; zones set
    before the run, changed from a developed state (the outflow velocities are re-published with buoyancy AND damping in the
    local macros), switched off; the time mean; rho, u, theta against the oracle."""
    nx, ny, nz = 52, 14, 12
    hm = np.zeros((ny, nx), np.int32); hm[3:8, 14:20] = 5; hm[8:12, 30:36] = 3
    sim, o, prof, thb = open_pair(B, nx, ny, nz, faces, hm, fp64, seed=3, want_mean=True, inplace=inplace)
    target = np.stack([prof, 0.1 * prof, np.zeros(nz)])
    tol = TOL64 if fp64 else TOL32
    for obj in (o, sim):
        obj.set_damping((4, 8, 3, 3, 0, 5), (0.05, 0.2, 0.05, 0.05, 0.0, 0.3), target)
        obj.mean_config(10, 5)
    sim.step(61); o.step(61)
    e_flow, e_th = errs(sim, o, 1.0)
    assert e_flow <= tol and e_th <= tol, ("zones", faces, fp64, e_flow, e_th)
    gm = sim.get_mean(f64=True); om = o.get_mean()
    assert gm[3] == om[3] == 11
    assert max(float(np.abs(a.cpu().numpy() - b).max()) for a, b in zip(gm[:3], om[:3])) <= tol
    for obj in (o, sim):
        obj.set_damping((0, 12, 0, 0, 0, 3), (0.0, 0.4, 0.0, 0.0, 0.0, 0.1), target)
    e_flow, e_th = errs(sim, o, 1.0)
    assert e_flow <= tol and e_th <= tol
    sim.step(30); o.step(30)
    e_flow, e_th = errs(sim, o, 1.0)
    assert e_flow <= tol and e_th <= tol, ("changed", faces, fp64, e_flow, e_th)
    for obj in (o, sim):
        obj.set_damping([0] * 6, [0.0] * 6, None)
    sim.step(20); o.step(20)
    e_flow, e_th = errs(sim, o, 1.0)
    assert e_flow <= tol and e_th <= tol, ("off", faces, fp64, e_flow, e_th)
    # the zones matter: the same run without them differs
    sim2, o2, _, _ = open_pair(B, nx, ny, nz, faces, hm, fp64, seed=3)
    o2.step(111)
    assert max(float(np.abs(a - b).max()) for a, b in zip(o.get_macros(), o2.get_macros())) > 1e-4
    sim.close(); o.close(); sim2.close(); o2.close()


def test_uniformly_warm_damped_box_settles_at_a_over_sigma_on_the_gpu(B):
    """The closed form that pins the oracle (w* = w_t + g beta dtheta / sigma, defect x (1 - sigma/2)/(1 + sigma/2) per step), on
    the FP32 path itself."""
    nx, ny, nz = 40, 6, 2
    sigma, gbeta, dth, wt, w0 = 0.25, 2e-4, 1.5, 0.01, 0.03
    sim = B.Lbm(nx, ny, nz, 5e-3, 0.1, 0.0, (0, 0, 0), [P] * 6)
    sim.set_flags(None)
    ut = np.zeros((3, nz)); ut[2] = wt
    sim.set_damping((0, 0, 0, 0, 1, 1), (0, 0, 0, 0, sigma, sigma), ut)
    sim.set_thermal(0.02, gbeta, 300.0)
    sim.set_macros(None, None, None, np.full((nz, ny, nx), w0, dtype=np.float32))
    sim.set_theta(np.full((nz, ny, nx), 300.0 + dth), f64=True)
    a, q = gbeta * dth, (1 - sigma / 2) / (1 + sigma / 2)
    wstar = wt + a / sigma
    w1 = (w0 + a / 2 + sigma / 2 * wt) / (1 + sigma / 2)
    for k in (1, 2, 10, 40):
        sim.step(k - sim.get_step())
        uz = sim.get_macros()[3].cpu().numpy()
        assert np.abs(uz - (wstar + (w1 - wstar) * q ** (k - 1))).max() < 2e-7, k
    sim.close()


@pytest.mark.parametrize("inplace", [False, True])
@pytest.mark.parametrize("fp64", [False, True])
def test_whole_open_boundary_stack_on_a_thermal_run(B, fp64, inplace):
    """Everything PAPER.md:175 / Table 1 lists, at once: equilibrium velocity faces with a warm inflow, the
    global flux correction, sponge + buffer nudging, synthetic fluctuations on the active inflow cells — whose thermal state
    follows the same velocity (reading 28) — buoyancy, LES, Coriolis, the time mean.  Fluctuations switched on before the
    thermal lattice and after it, theta_b changed while they run, a second mode table from a developed state, off again."""
    from paper_2607_04516_b200 import workloads as Wl
    nx, ny, nz = 48, 20, 12
    hm = np.zeros((ny, nx), np.int32); hm[5:10, 14:20] = 5; hm[11:15, 30:36] = 3
    faces = (EQF, EQO, EQF, EQF, W, EQF)
    modes = Wl.inflow_modes(32, 41, 2 * np.pi / 30, np.pi, convect=(0.05, 0.01, 0.0))
    tol = TOL64 if fp64 else TOL32
    for order in ("turbulence first", "thermal first"):
        from oracle import Oracle
        prof = (0.05 * np.log((np.arange(nz) + 0.5) / 0.1) / np.log(nz / 0.1)).clip(0)
        thb = 1.0 + 0.4 * np.exp(-np.arange(nz) / 4.0)
        u0 = np.broadcast_to(prof[:, None, None], (nz, ny, nx)).copy()
        th0 = 1.0 + 0.05 * np.random.default_rng(8).standard_normal((nz, ny, nx))
        target = np.stack([prof, 0.1 * prof, np.zeros(nz)])
        args = (nx, ny, nz, 3e-3, 0.1, 1e-3, (0.0, 0, 0), faces)
        o = Oracle(*args)
        sim = B.Lbm(*args, fp64=fp64, want_mean=True, inplace=inplace)
        for obj, kw in ((o, {}), (sim, {"f64": True})):
            obj.set_flags(hm)
            obj.set_inlet_profile(prof, 0.1 * prof, None, **kw)
            obj.set_macros(None, u0, None, None, **kw)
            obj.balance_flux()
            obj.set_damping((4, 8, 3, 3, 0, 5), (0.05, 0.2, 0.05, 0.05, 0.0, 0.3), target)
            if order == "turbulence first":
                obj.set_inflow_turbulence(modes, 0.004, 2 * np.pi / 12, 2.5)
            obj.set_thermal(0.02, 3e-4, 1.0)
            obj.set_inlet_theta(thb, **kw)
            obj.set_theta(th0, u0, None, None, **kw)
            if order == "thermal first":
                obj.set_inflow_turbulence(modes, 0.004, 2 * np.pi / 12, 2.5)
            obj.mean_config(10, 5)
        e_flow, e_th = errs(sim, o, 1.0)
        assert e_flow <= tol and e_th <= tol, ("set-up", order, e_flow, e_th)
        sim.step(61); o.step(61)
        e_flow, e_th = errs(sim, o, 1.0)
        assert e_flow <= tol and e_th <= tol, (order, fp64, e_flow, e_th)
        gm = sim.get_mean(f64=True); om = o.get_mean()
        assert gm[3] == om[3] == 11
        assert max(float(np.abs(a.cpu().numpy() - b).max()) for a, b in zip(gm[:3], om[:3])) <= tol
        for obj, kw in ((o, {}), (sim, {"f64": True})):
            obj.set_inlet_theta(thb + 0.1, **kw)            # while the fluctuations run
            obj.set_inflow_turbulence(Wl.inflow_modes(9, 5, 0.2, 2.0, convect=(0.04, 0.0, 0.0)), 0.002, 0.3)
        e_flow, e_th = errs(sim, o, 1.0)
        assert e_flow <= tol and e_th <= tol
        sim.step(30); o.step(30)
        e_flow, e_th = errs(sim, o, 1.0)
        assert e_flow <= tol and e_th <= tol, ("second table", order, fp64, e_flow, e_th)
        for obj in (o, sim):
            obj.set_inflow_turbulence(None)
        sim.step(20); o.step(20)
        e_flow, e_th = errs(sim, o, 1.0)
        assert e_flow <= tol and e_th <= tol, ("off", order, fp64, e_flow, e_th)
        sim.close(); o.close()

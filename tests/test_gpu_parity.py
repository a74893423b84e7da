"""Parity of the CUDA path (through the C ABI) against the CPU FP64 oracle, on the same seeded inputs.

Bars (BASELINE.json north_star): flags and link classes bit-exact; max-abs(rho, u) <= 1e-5 (lattice units) after
100 steps for the FP32 path; the FP64 instantiation of the same kernels must agree to ~1e-12.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL32 = 1e-5    # north_star
TOL64 = 2e-12   # rounding order only


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2607_04516_b200 import binding, build
    build.build()
    return binding


def make_oracle(wl):
    from oracle import Oracle
    o = Oracle(wl.nx, wl.ny, wl.nz, wl.nu0, wl.Cs, wl.f_cor, wl.F, wl.faces)
    o.set_flags(wl.height)
    if wl.inlet_profile is not None:
        o.set_inlet_profile(*wl.inlet_profile)
    if wl.init is not None:
        o.set_macros(*wl.init)
    else:
        o.set_macros()
    return o


def max_err(sim, o, f64=False):
    g = [a.cpu().numpy() for a in sim.get_macros(f64=f64)]
    r = o.get_macros()
    assert all(np.isfinite(a).all() for a in g)
    return max(float(np.abs(a.astype(np.float64) - b).max()) for a, b in zip(g, r))


def check_flags_links(sim, o):
    np.testing.assert_array_equal(sim.get_flags(), o.get_flags())
    np.testing.assert_array_equal(sim.get_links(), o.get_links())


# ---------------------------------------------------------------------------------------------- integer work

FACE_SETS = [
    (0, 0, 0, 0, 0, 0), (3, 4, 0, 0, 1, 2), (3, 4, 2, 2, 1, 2), (3, 4, 3, 3, 1, 2), (0, 0, 0, 0, 1, 2),
    (1, 1, 1, 1, 1, 1), (2, 2, 2, 2, 2, 2), (2, 1, 0, 0, 2, 1), (4, 3, 1, 2, 0, 0),
    (3, 4, 2, 4, 1, 2),     # two EQ_OUTFLOW faces meet (DESIGN.md §4 reading 24)
]


@pytest.mark.parametrize("faces", FACE_SETS)
def test_flags_and_links_bit_exact_small_ragged_boxes(B, faces):
    from oracle import Oracle
    rng = np.random.default_rng(abs(hash(faces)) % (2 ** 32))
    for nx, ny, nz in [(6, 5, 4), (33, 7, 9), (70, 3, 5), (1, 1, 3), (5, 1, 1)]:
        hm = rng.integers(-1, nz + 2, size=(ny, nx)).astype(np.int32)
        hm[rng.random((ny, nx)) < 0.5] = 0
        o = Oracle(nx, ny, nz, 1e-3, 0.1, 0.0, (0, 0, 0), faces)
        o.set_flags(hm)
        sim = B.Lbm(nx, ny, nz, 1e-3, 0.1, 0.0, (0, 0, 0), faces)
        sim.set_flags(hm)
        check_flags_links(sim, o)
        sim.close()


def test_flags_and_links_bit_exact_config3_full(B):
    from paper_2607_04516_b200 import workloads as W
    from oracle import Oracle
    wl = W.config3()
    o = Oracle(wl.nx, wl.ny, wl.nz, wl.nu0, wl.Cs, wl.f_cor, wl.F, wl.faces)
    o.set_flags(wl.height)
    sim = B.Lbm(wl.nx, wl.ny, wl.nz, wl.nu0, wl.Cs, wl.f_cor, wl.F, wl.faces, want_mean=False)
    sim.set_flags(wl.height)
    check_flags_links(sim, o)
    assert int((sim.get_flags() == 1).sum()) == int(wl.height.sum())


def test_null_heightmap_is_flat_ground_and_device_heightmap_works(B):
    import torch
    from oracle import Oracle
    faces = (3, 4, 2, 2, 1, 2)
    o = Oracle(20, 10, 6, 1e-3, 0.1, 0.0, (0, 0, 0), faces)
    o.set_flags(None)
    sim = B.Lbm(20, 10, 6, 1e-3, 0.1, 0.0, (0, 0, 0), faces)
    sim.set_flags(None)
    check_flags_links(sim, o)
    hm = np.zeros((10, 20), dtype=np.int32)
    hm[3:6, 5:9] = 4
    o.set_flags(hm)
    sim.set_flags(torch.from_numpy(hm).cuda())
    check_flags_links(sim, o)


# ---------------------------------------------------------------------------------------------- floating point

def test_config1_100_and_200_steps(B):
    from paper_2607_04516_b200 import workloads as W
    wl = W.config1()
    o = make_oracle(wl)
    sim = B.from_workload(wl)
    check_flags_links(sim, o)
    for upto in (100, 200):
        o.step(upto - o.get_step())
        sim.step(upto - sim.get_step())
        e = max_err(sim, o)
        print(f"C1 step {upto}: max|gpu32 - oracle| = {e:.3e}")
        assert e <= TOL32
    assert sim.get_step() == 200


def test_config1_fp64_kernels_agree_to_rounding(B):
    from paper_2607_04516_b200 import workloads as W
    wl = W.config1()
    o = make_oracle(wl)
    sim = B.from_workload(wl, fp64=True)
    o.step(100)
    sim.step(100)
    e = max_err(sim, o, f64=True)
    print(f"C1 step 100: max|gpu64 - oracle| = {e:.3e}")
    assert e <= TOL64


@pytest.mark.parametrize("Cs", [0.0, 0.1])
def test_config2_taylor_green_100_steps(B, Cs):
    from paper_2607_04516_b200 import workloads as W
    wl = W.config2(Cs=Cs)
    o = make_oracle(wl)
    sim = B.from_workload(wl)
    o.step(100)
    sim.step(100)
    e = max_err(sim, o)
    print(f"C2 Cs={Cs} step 100: max|gpu32 - oracle| = {e:.3e}")
    assert e <= TOL32


def test_config3_full_100_steps(B):
    """The bench workload itself, in the launch configuration bench.py times, against the oracle on every cell."""
    from paper_2607_04516_b200 import workloads as W
    wl = W.config3()
    o = make_oracle(wl)
    sim = B.from_workload(wl, want_mean=False)
    o.step(100)
    sim.step(100)
    e = max_err(sim, o)
    print(f"C3 400x400x100 step 100: max|gpu32 - oracle| = {e:.3e}")
    assert e <= TOL32


def test_config3_crop_fp64_and_ragged_sizes(B):
    from paper_2607_04516_b200 import workloads as W
    wl = W.config3(nx=150, ny=77, nz=50)   # 150 and 77 are not multiples of the warp or of 4
    o = make_oracle(wl)
    s32 = B.from_workload(wl)
    s64 = B.from_workload(wl, fp64=True)
    o.step(100)
    s32.step(100)
    s64.step(100)
    e32, e64 = max_err(s32, o), max_err(s64, o, f64=True)
    print(f"C3 crop step 100: fp32 {e32:.3e}  fp64 {e64:.3e}")
    assert e32 <= TOL32 and e64 <= TOL64


def test_config4_crop_veering_inlet_on_three_faces(B):
    from paper_2607_04516_b200 import workloads as W
    wl = W.config4(nx=120, ny=90, nz=200)
    o = make_oracle(wl)
    sim = B.from_workload(wl)
    check_flags_links(sim, o)
    o.step(100)
    sim.step(100)
    e = max_err(sim, o)
    print(f"C4 crop step 100: {e:.3e}")
    assert e <= TOL32


def test_config5_precursor_crop_with_pressure_gradient_force(B):
    from paper_2607_04516_b200 import workloads as W
    wl = W.config5_precursor(nx=64, ny=48, nz=200)
    o = make_oracle(wl)
    sim = B.from_workload(wl)
    o.step(100)
    sim.step(100)
    e = max_err(sim, o)
    print(f"C5 precursor crop step 100: {e:.3e}")
    assert e <= TOL32


def test_config5_chain_precursor_plane_feeds_main_inlet_every_step(B):
    """Coupled run (a8): each step the precursor plane x_s is written into the main x- inlet, then both advance.
    The oracle side does the same through get_macros/set_inlet_plane."""
    from paper_2607_04516_b200 import workloads as W
    from oracle import Oracle
    pre = W.config5_precursor(nx=32, ny=24, nz=40)
    main = W.config5_main(nx=96, ny=60, nz=40)   # 60 is not a multiple of 24: the last tile is cut
    xs = 16
    op, om = make_oracle(pre), make_oracle(main)
    gp, gm = B.from_workload(pre), B.from_workload(main)
    reps = -(-main.ny // pre.ny)
    for _ in range(30):
        _, ux, uy, uz = op.get_macros()
        plane = np.stack([np.tile(q[:, :, xs], (1, reps))[:, :main.ny] for q in (ux, uy, uz)])
        om.set_inlet_plane(0, plane)
        gm.feed_inlet(gp, xs)
        op.step(1); om.step(1)
        gp.step(1); gm.step(1)
    e_pre, e_main = max_err(gp, op), max_err(gm, om)
    print(f"C5 chain step 30: precursor {e_pre:.3e} main {e_main:.3e}")
    assert e_pre <= TOL32 and e_main <= TOL32


def test_config5_chain_on_two_streams_equals_the_chain_on_one(B):
    """lbm_feed_inlet with the precursor and the main lattice on different streams: the read of the plane waits for the
    precursor's last step, and the precursor's next steps wait for the read (its stream runs far ahead of the 7x larger
    main lattice otherwise and rewrites the buffer the plane lies in).  Bit-identical to the single-stream chain."""
    import torch
    from paper_2607_04516_b200 import workloads as W
    pre = W.config5_precursor(nx=32, ny=24, nz=40)
    main = W.config5_main(nx=224, ny=60, nz=40)
    xs = 16
    results = []
    for two in (False, True):
        sp = torch.cuda.Stream() if two else None
        sm = torch.cuda.Stream() if two else None
        torch.cuda.synchronize()
        gp, gm = B.from_workload(pre, stream=sp), B.from_workload(main, stream=sm)
        for _ in range(40):
            gm.feed_inlet(gp, xs)
            gp.step(1); gm.step(1)
        results.append([a.cpu().numpy() for a in gm.get_macros()] + [a.cpu().numpy() for a in gp.get_macros()])
        torch.cuda.synchronize()
        gp.close(); gm.close()
    for a, b in zip(*results):
        np.testing.assert_array_equal(a, b)


def test_inlet_plane_host_and_device_pointers(B):
    import torch
    from oracle import Oracle
    rng = np.random.default_rng(12)
    nx, ny, nz = 24, 10, 8
    faces = (3, 4, 3, 3, 1, 2)
    o = Oracle(nx, ny, nz, 2e-3, 0.1, 0.0, (0, 0, 0), faces)
    o.set_flags()
    sim = B.Lbm(nx, ny, nz, 2e-3, 0.1, 0.0, (0, 0, 0), faces)
    sim.set_flags()
    px = (0.03 + 0.01 * rng.random((3, nz, ny))).astype(np.float32)
    py = (0.03 + 0.01 * rng.random((3, nz, nx))).astype(np.float32)
    o.set_inlet_plane(0, px); o.set_inlet_plane(2, py); o.set_inlet_plane(3, py)
    sim.set_inlet_plane(0, px)                             # host pointer
    sim.set_inlet_plane(2, torch.from_numpy(py).cuda())    # device pointer
    sim.set_inlet_plane(3, py.astype(np.float64), f64=True)
    o.set_macros(None, np.full(o.shape, 0.03), np.full(o.shape, 0.03), None)
    sim.set_macros(None, np.full(o.shape, 0.03, dtype=np.float32), np.full(o.shape, 0.03, dtype=np.float32), None)
    o.step(40); sim.step(40)
    assert max_err(sim, o) <= TOL32


def test_time_mean_matches_oracle_and_fused_equals_standalone_definition(B):
    from paper_2607_04516_b200 import workloads as W
    wl = W.config3(nx=96, ny=64, nz=40)
    o = make_oracle(wl)
    sim = B.from_workload(wl)
    o.mean_config(20, 5); sim.mean_config(20, 5)
    o.step(60); sim.step(60)
    gm = sim.get_mean()
    om = o.get_mean()
    assert gm[3] == om[3] == 9
    for a, b in zip(gm[:3], om[:3]):
        assert float(np.abs(a.cpu().numpy() - b).max()) <= TOL32
    flags = sim.get_flags()
    assert np.all(gm[0].cpu().numpy()[flags == 1] == 0)
    # horizontal mean profile within 1e-5 as well
    pg = W.mean_profile(gm[0].cpu().numpy(), flags)
    po = W.mean_profile(om[0], flags)
    assert np.abs(pg - po).max() <= TOL32
    sim.mean_reset()
    assert sim.get_mean()[3] == 0


def test_state_roundtrip_and_restart_from_a_developed_gpu_state(B):
    """lbm_get_state at a developed step -> the oracle continues 100 steps from that state."""
    from paper_2607_04516_b200 import workloads as W
    wl = W.config1()
    sim = B.from_workload(wl)
    sim.step(700)
    st = sim.get_state(out="host")
    assert np.isfinite(st).all()
    o = make_oracle(wl)
    o.set_state(st)
    o.set_step(700)
    assert max_err(sim, o) <= 1e-7          # same state, FP32 vs FP64 evaluation of the macros
    o.step(100); sim.step(100)
    e = max_err(sim, o)
    print(f"C1 restart 700 -> 800: {e:.3e}")
    assert e <= TOL32
    # round trip through set_state is the identity on the FP32 state
    sim2 = B.from_workload(wl)
    sim2.set_state(sim.get_state())
    a, b = sim.get_state(out="host"), sim2.get_state(out="host")
    assert np.array_equal(a, b)


def test_rest_state_is_exactly_zero_in_shifted_storage(B):
    hm = np.zeros((12, 16), dtype=np.int32)
    hm[3:6, 4:8] = 5
    _, w, _ = __import__("oracle").lattice()
    for faces in [(3, 4, 0, 0, 1, 2), (2, 2, 1, 1, 0, 0), (0,) * 6]:
        sim = B.Lbm(16, 12, 8, 1e-3, 0.1, 0.0, (0, 0, 0), faces)
        sim.set_flags(hm)
        sim.set_inlet_profile(np.zeros(8, dtype=np.float32))
        sim.set_macros()
        sim.step(50)
        st = sim.get_state(out="host")
        assert np.array_equal(st, np.broadcast_to(w[:, None, None, None], st.shape))
        rho, ux, uy, uz = (a.cpu().numpy() for a in sim.get_macros())
        assert np.all(rho == 1) and np.all(ux == 0) and np.all(uy == 0) and np.all(uz == 0)


def test_mass_conservation_and_inertial_rotation_on_the_gpu(B):
    """Properties that hold at any size, checked on the FP32 path itself: periodic-box mass is conserved to FP32
    rounding and total momentum turns by -2 atan(f/2) per step."""
    import math
    import torch
    from paper_2607_04516_b200 import workloads as W
    wl = W.config2(Cs=0.1, n=64, nz=16)
    wl.f_cor = 0.01
    sim = B.from_workload(wl)
    c, _ = B.lattice()
    ct = torch.tensor(c, dtype=torch.float64, device="cuda")

    def mom():
        st = sim.get_state()
        return torch.einsum("ia,izyx->a", ct, st).cpu().numpy(), float(st.sum())

    P0, m0 = mom()
    sim.step(200)
    P1, m1 = mom()
    assert abs(m1 / m0 - 1) < 1e-7
    assert abs(np.hypot(*P1[:2]) / np.hypot(*P0[:2]) - 1) < 1e-4   # FP32 rounding over 200 steps (FP64 oracle: 1e-12)
    dth = math.atan2(P1[1], P1[0]) - math.atan2(P0[1], P0[0])
    assert dth == pytest.approx(-200 * 2 * math.atan(0.005), abs=1e-4)


def test_zero_steps_and_call_order_errors(B):
    sim = B.Lbm(8, 8, 8, 1e-3)
    with pytest.raises(B.LbmError, match="LBM_ESTATE"):
        sim.step(1)
    with pytest.raises(B.LbmError, match="LBM_ESTATE"):
        sim.set_macros()
    with pytest.raises(B.LbmError, match="LBM_EINVAL"):
        sim.set_boundaries((0, 1, 0, 0, 0, 0))
    sim.set_flags()
    sim.set_macros()
    n0 = sim.launch_count()
    sim.step(0)
    assert sim.get_step() == 0 and sim.launch_count() == n0
    with pytest.raises(B.LbmError, match="LBM_EINVAL"):
        sim.step(-1)
    nomean = B.Lbm(8, 8, 8, 1e-3, want_mean=False)
    with pytest.raises(B.LbmError, match="LBM_ESTATE"):
        nomean.mean_config(0, 1)


def test_host_pointer_getters_equal_device_pointer_getters(B):
    from paper_2607_04516_b200 import workloads as W
    sim = B.from_workload(W.config1())
    sim.step(10)
    dev = [a.cpu().numpy() for a in sim.get_macros()]
    host = sim.get_macros(out="host")
    for a, b in zip(dev, host):
        assert np.array_equal(a, b)


# ---------------------------------------------------------------------------------------------- kernel variants

@pytest.mark.parametrize("variant", [0, 1, 2, 3])     # every launch shape lbm_set_variant offers (include/lbm.h)
@pytest.mark.parametrize("shape", [(37, 11, 9), (64, 36, 20), (130, 50, 7), (132, 9, 6), (4, 5, 6), (8, 3, 3)])
def test_every_step_kernel_variant_matches_the_oracle(B, variant, shape):
    """One cell per thread, 2 and 4 x-cells per thread with 64 / 128-bit accesses, and the cooperative multi-step launch
    compute the same step: ragged boxes (fall back to one cell per thread), nx % 4 == 0 and nx % 2 == 0 boxes, rows
    shorter than a warp (several rows per warp, shuffles across row ends), a last warp that is partly beyond the plane,
    buildings, every face rule, forcing, mean sampling."""
    from oracle import Oracle
    nx, ny, nz = shape
    rng = np.random.default_rng(nx * 1000 + ny)
    hm = np.zeros((ny, nx), dtype=np.int32)
    for _ in range(6):
        x0, y0 = int(rng.integers(0, max(nx - 6, 1))), int(rng.integers(0, max(ny - 3, 1)))
        hm[y0:y0 + 3, x0:x0 + 4] = int(rng.integers(1, nz))
    prof = (0.05 * np.log((np.arange(nz) + 0.5) / 0.1) / np.log(nz / 0.1)).clip(0).astype(np.float32)
    for faces in [(3, 4, 0, 0, 1, 2), (3, 4, 2, 2, 1, 2), (0, 0, 0, 0, 1, 2), (3, 4, 3, 3, 1, 2), (3, 4, 2, 4, 1, 2)]:
        args = (nx, ny, nz, 2e-3, 0.1, 1e-3, (1e-6, 0, 0), faces)
        o = Oracle(*args)
        o.set_flags(hm)
        o.set_inlet_profile(prof.astype(np.float64), 0.1 * prof.astype(np.float64), None)
        ux0 = np.broadcast_to(prof[:, None, None], (nz, ny, nx)).astype(np.float32).copy()
        o.set_macros(None, ux0.astype(np.float64), None, None)
        o.mean_config(10, 5)
        sim = B.Lbm(*args)
        sim.set_variant(variant)
        sim.set_flags(hm)
        sim.set_inlet_profile(prof, 0.1 * prof, None)
        sim.set_macros(None, ux0, None, None)
        sim.mean_config(10, 5)
        o.step(40)
        sim.step(40)
        e = max_err(sim, o)
        assert e <= TOL32, (variant, shape, faces, e)
        *gm, n = sim.get_mean()
        *om, on = o.get_mean()
        assert n == on == 7
        em = max(float(np.abs(a.cpu().numpy().astype(np.float64) - b).max()) for a, b in zip(gm, om))
        assert em <= TOL32, (variant, shape, faces, em)
        sim.close()


# ---------------------------------------------------------------------------------------------- full Coriolis vector

@pytest.mark.parametrize("fp64", [False, True])
def test_full_coriolis_vector_matches_the_oracle(B, fp64):
    """PAPER.md:61 / Table 1: full rotation vector through Guo forcing.  Tilted axis, buildings, every face
    rule, forcing, LES; 100 steps; FP32 within 1e-5, FP64 within rounding order."""
    from oracle import Oracle
    nx, ny, nz = 48, 40, 24
    rng = np.random.default_rng(77)
    hm = np.zeros((ny, nx), dtype=np.int32)
    for _ in range(5):
        x0, y0 = int(rng.integers(4, nx - 10)), int(rng.integers(0, ny - 4))
        hm[y0:y0 + 4, x0:x0 + 5] = int(rng.integers(1, nz - 4))
    prof = (0.05 * np.log((np.arange(nz) + 0.5) / 0.1) / np.log(nz / 0.1)).clip(0)
    fv = (1.5e-3, -1.0e-3, 2.0e-3)
    for faces in [(3, 4, 2, 2, 1, 2), (0, 0, 0, 0, 1, 2)]:
        args = (nx, ny, nz, 2e-3, 0.1, 5e-4, (1e-6, -5e-7, 0.0), faces)
        o = Oracle(*args)
        o.set_coriolis(fv)
        o.set_flags(hm)
        o.set_inlet_profile(prof, 0.2 * prof, None)
        ux0 = np.broadcast_to(prof[:, None, None], (nz, ny, nx)).copy()
        o.set_macros(None, ux0, None, None)
        sim = B.Lbm(*args, fp64=fp64)
        sim.set_coriolis(fv)
        sim.set_flags(hm)
        sim.set_inlet_profile(prof, 0.2 * prof, None, f64=True)
        sim.set_macros(None, ux0, None, None, f64=True)
        o.step(100)
        sim.step(100)
        e = max_err(sim, o, f64=fp64)
        assert e <= (TOL64 if fp64 else TOL32), (faces, fp64, e)
        sim.close()


def test_momentum_turns_about_a_tilted_axis_on_the_fp32_path(B):
    """Closed form on the GPU path itself: periodic box, total momentum turns about f by 2 atan(|f|/2) per step."""
    n = 32
    fv = np.array([2e-3, -1e-3, 2.5e-3])
    sim = B.Lbm(n, n, n, 5e-3, 0.1, 0.0, (0, 0, 0), (0, 0, 0, 0, 0, 0), fp64=True)
    sim.set_coriolis(fv)
    sim.set_flags(None)
    x = np.arange(n) * 2 * np.pi / n
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    sim.set_macros(None, 0.03 + 0.01 * np.sin(Y), -0.02 + 0.01 * np.cos(Z), 0.015 + 0.01 * np.sin(X + Y), f64=True)
    c, opp = B.lattice()

    def P():
        f = sim.get_state().cpu().numpy()
        return np.array([(c[:, a][:, None, None, None] * f).sum() for a in range(3)])
    P0 = P()
    k = 40
    sim.step(k)
    Pk = P()
    axis = fv / np.linalg.norm(fv)
    th = -2.0 * np.arctan(0.5 * np.linalg.norm(fv)) * k
    K = np.array([[0, -axis[2], axis[1]], [axis[2], 0, -axis[0]], [-axis[1], axis[0], 0]])
    R = np.eye(3) + np.sin(th) * K + (1 - np.cos(th)) * (K @ K)
    assert np.abs(Pk - R @ P0).max() < 1e-10 * n ** 3
    sim.close()


# ---------------------------------------------------------------------------------------------- flux balancing

@pytest.mark.parametrize("fp64", [False, True])
@pytest.mark.parametrize("faces", [(3, 3, 3, 3, 1, 3), (3, 4, 3, 3, 1, 2), (3, 3, 0, 0, 1, 2)])
def test_flux_balancing_matches_the_oracle(B, faces, fp64):
    """PAPER.md:55 / :175: global flux-balancing correction over the open (EQ_FIXED) faces, then 50 steps."""
    from oracle import Oracle
    nx, ny, nz = 37, 22, 14
    rng = np.random.default_rng(11)
    hm = np.zeros((ny, nx), dtype=np.int32)
    hm[3:6, 0:3] = 5           # a building standing in the x- face
    hm[10:14, 15:20] = 9
    args = (nx, ny, nz, 5e-3, 0.1, 1e-3, (0.0, 0.0, 0.0), faces)
    o = Oracle(*args)
    sim = B.Lbm(*args, fp64=fp64)
    o.set_flags(hm)
    sim.set_flags(hm)
    for k in range(6):
        if faces[k] == 3:
            axis = k // 2
            n1 = ny if axis == 0 else nx
            n2 = ny if axis == 2 else nz
            pl = (0.03 * rng.standard_normal((3, n2, n1))).astype(np.float32).astype(np.float64)
            o.set_inlet_plane(k, pl)
            sim.set_inlet_plane(k, pl, f64=True)
    o.set_macros()
    sim.set_macros()
    ob, oa = o.balance_flux()
    gb, ga = sim.balance_flux()
    assert gb == pytest.approx(ob, rel=1e-6 if not fp64 else 1e-12, abs=1e-9)
    assert abs(oa) < 1e-12 and abs(ga) < (1e-12 if fp64 else 2e-5)
    assert max_err(sim, o, f64=fp64) <= (TOL64 if fp64 else 1e-7)
    o.step(50)
    sim.step(50)
    assert max_err(sim, o, f64=fp64) <= (TOL64 if fp64 else TOL32)
    sim.close()


# ---------------------------------------------------------------------------------------------- damping zones

@pytest.mark.parametrize("fp64", [False, True])
def test_damping_zones_match_the_oracle(B, fp64):
    """PAPER.md:175 / Table 1: top sponge + lateral buffer nudging towards the target boundary state.
    Buildings, veering inlet on three faces + outflow (the paper's open-face set-up) and a periodic variant, Coriolis
    vector, forcing, LES, zones on five faces with different widths / peaks; 100 steps; FP32 within 1e-5, FP64 within
    rounding order; macros taken inside the zones (the inversion carries sigma) and the fused time mean."""
    from oracle import Oracle
    nx, ny, nz = 50, 42, 24
    rng = np.random.default_rng(91)
    hm = np.zeros((ny, nx), dtype=np.int32)
    for _ in range(5):
        x0, y0 = int(rng.integers(10, nx - 14)), int(rng.integers(8, ny - 12))
        hm[y0:y0 + 4, x0:x0 + 5] = int(rng.integers(1, nz - 8))
    prof = (0.05 * np.log((np.arange(nz) + 0.5) / 0.1) / np.log(nz / 0.1)).clip(0)
    target = np.stack([prof, 0.2 * prof, np.zeros(nz)])
    width, peak = (6, 9, 5, 5, 0, 7), (0.05, 0.2, 0.1, 0.1, 0.0, 0.3)
    fv = (1.0e-3, -0.5e-3, 2.0e-3)
    for faces in [(3, 4, 3, 3, 1, 2), (0, 0, 0, 0, 1, 2)]:
        args = (nx, ny, nz, 2e-3, 0.1, 0.0, (1e-6, -5e-7, 0.0), faces)
        o = Oracle(*args)
        o.set_coriolis(fv)
        o.set_flags(hm)
        o.set_inlet_profile(prof, 0.2 * prof, None)
        ux0 = np.broadcast_to((0.8 * prof)[:, None, None], (nz, ny, nx)).copy()   # off target: the zones act from step 1
        o.set_macros(None, ux0, None, None)
        o.set_damping(width, peak, target)
        o.mean_config(50, 10)
        sim = B.Lbm(*args, fp64=fp64)
        sim.set_coriolis(fv)
        sim.set_flags(hm)
        sim.set_inlet_profile(prof, 0.2 * prof, None, f64=True)
        sim.set_macros(None, ux0, None, None, f64=True)
        sim.set_damping(width, peak, target)
        sim.mean_config(50, 10)
        # the zones must matter at the parity bar, or this test proves nothing
        ref = Oracle(*args)
        ref.set_coriolis(fv); ref.set_flags(hm); ref.set_inlet_profile(prof, 0.2 * prof, None); ref.set_macros(None, ux0, None, None)
        o.step(100)
        ref.step(100)
        sim.step(100)
        assert max(np.abs(a - b).max() for a, b in zip(o.get_macros(), ref.get_macros())) > 1e-3
        e = max_err(sim, o, f64=fp64)
        assert e <= (TOL64 if fp64 else TOL32), (faces, fp64, e)
        gm = sim.get_mean(f64=fp64)
        om = o.get_mean()
        assert gm[3] == om[3] == 6
        em = max(float(np.abs(a.cpu().numpy().astype(np.float64) - b).max()) for a, b in zip(gm[:3], om[:3]))
        assert em <= (TOL64 if fp64 else TOL32), (faces, fp64, em)
        # switching the zones off returns to the plain kernel: it follows the undamped oracle from the same state
        sim.set_damping((0,) * 6, (0,) * 6, None)
        o.set_damping((0,) * 6, (0,) * 6, None)
        o.step(20)
        sim.step(20)
        e = max_err(sim, o, f64=fp64)
        assert e <= (TOL64 if fp64 else TOL32), (faces, fp64, e)
        sim.close()


def test_uniform_zone_decays_by_the_trapezoidal_factor_on_the_fp32_path(B):
    """The closed form that pins the oracle, checked on the GPU path itself: two-layer free-slip slab, width-1 zones on
    z- and z+ (uniform sigma), uniform flow: u_k - u_t = (u_0 - u_t) q^(k-1) / (1 + sigma/2), q = (1 - s/2)/(1 + s/2)."""
    nx, ny, nz, sigma = 40, 9, 2, 0.2
    sim = B.Lbm(nx, ny, nz, 1e-2, 0.1, 0.0, (0, 0, 0), (0, 0, 0, 0, 2, 2))
    sim.set_flags(None)
    ut = np.zeros((3, nz)); ut[0] = 0.03; ut[1] = -0.01
    sim.set_damping((0, 0, 0, 0, 1, 1), (0, 0, 0, 0, sigma, sigma), ut)
    u0 = np.array([0.08, 0.02])
    sim.set_macros(None, np.full((nz, ny, nx), u0[0]), np.full((nz, ny, nx), u0[1]), None, f64=True)
    q = (1 - sigma / 2) / (1 + sigma / 2)
    for k in (1, 2, 10, 30):
        sim.step(k - sim.get_step())
        r, ux, uy, uz = [a.cpu().numpy().astype(np.float64) for a in sim.get_macros()]
        assert np.abs(ux - (ut[0, 0] + (u0[0] - ut[0, 0]) * q ** (k - 1) / (1 + sigma / 2))).max() < 2e-7
        assert np.abs(uy - (ut[1, 0] + (u0[1] - ut[1, 0]) * q ** (k - 1) / (1 + sigma / 2))).max() < 2e-7
        assert np.abs(r - 1).max() < 1e-6 and np.abs(uz).max() < 1e-7
    sim.close()


def test_set_damping_argument_errors(B):
    sim = B.Lbm(8, 8, 8, 1e-2, 0.1, 0.0, (0, 0, 0), (0, 0, 0, 0, 1, 2))
    sim.set_flags(None)
    with pytest.raises(B.LbmError):
        sim.set_damping((1,) * 6, (1.5,) * 6, np.zeros((3, 8)))
    with pytest.raises(B.LbmError):
        sim.set_damping((-1, 0, 0, 0, 0, 0), (0.1,) * 6, np.zeros((3, 8)))
    with pytest.raises(B.LbmError):
        sim.set_damping((2,) * 6, (0.1,) * 6, None)
    sim.set_damping((0,) * 6, (0.5,) * 6, None)   # off: target not needed
    sim.step(2)
    sim.close()


# ---------------------------------------------------------------------------------------------- synthetic inflow fluctuations

@pytest.mark.parametrize("fp64", [False, True])
def test_inflow_fluctuations_match_the_oracle(B, fp64):
    """PAPER.md:160 / Table 1: synthetic von Karman fluctuations on active inflow cells.  The paper's open-face
    set-up (veering mean on three EQ_FIXED faces + outflow: x- and y- see inflow, y+ outflow), buildings, LES, 64 modes
    carried with the reference wind; switched on at step 0 and again from a developed state (t = 37), 100 steps;
    FP32 within 1e-5, FP64 within rounding order; then switched off: the mean returns."""
    from oracle import Oracle
    from paper_2607_04516_b200 import workloads as W
    nx, ny, nz = 50, 42, 24
    rng = np.random.default_rng(17)
    hm = np.zeros((ny, nx), dtype=np.int32)
    for _ in range(5):
        x0, y0 = int(rng.integers(10, nx - 14)), int(rng.integers(8, ny - 12))
        hm[y0:y0 + 4, x0:x0 + 5] = int(rng.integers(1, nz - 8))
    prof = (0.05 * np.log((np.arange(nz) + 0.5) / 0.1) / np.log(nz / 0.1)).clip(0)
    modes = W.inflow_modes(64, 23, 2 * np.pi / 40, np.pi, convect=(0.05, 0.01, 0.0))
    u_rms, k_e, k_eta = 0.004, 2 * np.pi / 15, 2.5
    args = (nx, ny, nz, 2e-3, 0.1, 1e-4, (0.0, 0.0, 0.0), (3, 4, 3, 3, 1, 2))
    ux0 = np.broadcast_to(prof[:, None, None], (nz, ny, nx)).copy()
    uy0 = 0.2 * ux0

    def setup(obj, f64kw):
        obj.set_flags(hm)
        obj.set_inlet_profile(prof, 0.2 * prof, None, **f64kw)
        obj.set_macros(None, ux0, uy0, None, **f64kw)

    o = Oracle(*args)
    setup(o, {})
    sim = B.Lbm(*args, fp64=fp64)
    setup(sim, {"f64": True})
    tol = TOL64 if fp64 else TOL32
    o.set_inflow_turbulence(modes, u_rms, k_e, k_eta)
    sim.set_inflow_turbulence(modes, u_rms, k_e, k_eta)
    assert max_err(sim, o, f64=fp64) <= tol            # the inflow cells at t = 0
    ref = Oracle(*args)
    setup(ref, {})
    for upto in (37, 100):
        o.step(upto - o.get_step())
        sim.step(upto - sim.get_step())
        e = max_err(sim, o, f64=fp64)
        assert e <= tol, (upto, fp64, e)
    ref.step(100)
    assert max(np.abs(a - b).max() for a, b in zip(o.get_macros(), ref.get_macros())) > 2e-3   # the fluctuations matter
    # mean-changing calls are refused while the fluctuations ride on it
    with pytest.raises(B.LbmError):
        sim.set_inlet_profile(prof, None, None, f64=True)
    with pytest.raises(B.LbmError):
        sim.balance_flux()
    # a different table from a developed state
    modes2 = W.inflow_modes(17, 5, 0.2, 2.0, convect=(0.04, 0.0, 0.0))
    o.set_inflow_turbulence(modes2, 0.002, 0.3)
    sim.set_inflow_turbulence(modes2, 0.002, 0.3)
    o.step(30)
    sim.step(30)
    assert max_err(sim, o, f64=fp64) <= tol
    # off: the boundary returns to the mean, and the plain path continues
    o.set_inflow_turbulence(None)
    sim.set_inflow_turbulence(None)
    fl = o.get_flags()
    g = [a.cpu().numpy().astype(np.float64) for a in sim.get_macros(f64=fp64)]
    assert np.abs(g[1][fl == 2] - ux0[fl == 2]).max() < 1e-7 and np.abs(g[2][fl == 2] - uy0[fl == 2]).max() < 1e-7
    o.step(20)
    sim.step(20)
    assert max_err(sim, o, f64=fp64) <= tol
    sim.set_inlet_profile(prof, 0.2 * prof, None, f64=True)    # allowed again
    sim.close()


@pytest.mark.parametrize("fp64", [False, True])
def test_active_inflow_threshold_is_decided_like_the_oracle(B, fp64):
    """DESIGN.md §4 reading 21: active inflow <=> ub.n < -1e-7, compared in FP64 on both sides.  One x- face whose mean
    normal components straddle the constant — 5e-8 and the float32 just below 1e-7 keep the mean, the float32 just above
    1e-7 (= float32(1e-7)) and 2e-7 fluctuate; the inputs are float32-representable, so the FP32 handle stores exactly
    what the oracle gets.  Mirror of tests/test_oracle_inflow.py::test_active_inflow_threshold_..."""
    from oracle import Oracle
    from paper_2607_04516_b200 import workloads as W
    nx, ny, nz = 8, 8, 4
    above = np.float32(1e-7)
    assert float(above) > 1e-7
    below = np.nextafter(above, np.float32(0))
    assert float(below) < 1e-7
    un = np.array([5e-8, float(below), float(above), 2e-7, -2e-7, 1e-6, 0.0, -5e-8], dtype=np.float32).astype(np.float64)
    active = np.array([False, False, True, True, False, True, False, False])
    plane = np.zeros((3, nz, ny))
    plane[0] = un[None, :]
    plane[1] = 0.0078125
    args = (nx, ny, nz, 1e-2, 0.0, 0.0, (0, 0, 0), (3, 4, 0, 0, 2, 2))
    o = Oracle(*args); o.set_flags(None); o.set_inlet_plane(0, plane); o.set_macros()
    sim = B.Lbm(*args, fp64=fp64); sim.set_flags(None); sim.set_inlet_plane(0, plane, f64=True); sim.set_macros()
    modes = W.inflow_modes(8, 21, 0.2, 2.0)
    o.set_inflow_turbulence(modes, 0.01, 0.5)
    sim.set_inflow_turbulence(modes, 0.01, 0.5)
    for _ in range(3):
        g = [a.cpu().numpy().astype(np.float64) for a in sim.get_macros(f64=fp64)]
        dev = np.sqrt((g[1][:, :, 0] - un[None, :]) ** 2 + (g[2][:, :, 0] - 0.0078125) ** 2 + g[3][:, :, 0] ** 2)
        assert dev[:, ~active].max() < 1e-9 and dev[:, active].min() > 1e-4
        assert max_err(sim, o, f64=fp64) <= (TOL64 if fp64 else TOL32)
        o.step(1); sim.step(1)
    sim.close()


def test_inflow_fluctuation_phase_stays_exact_at_large_step_numbers(B):
    """t ~ 1e5 steps: the FP64 phase reduction keeps the FP32 path on the oracle (an FP32 phase would be off by ~1e-3 rad)."""
    from oracle import Oracle
    from paper_2607_04516_b200 import workloads as W
    nx, ny, nz = 12, 40, 16
    args = (nx, ny, nz, 1e-2, 0.0, 0.0, (0, 0, 0), (3, 4, 0, 0, 1, 2))
    prof = np.full(nz, 0.05)
    modes = W.inflow_modes(32, 2, 0.2, 3.0, convect=(0.05, 0.02, 0.0))
    o = Oracle(*args)
    sim = B.Lbm(*args)
    for obj, kw in ((o, {}), (sim, {"f64": True})):
        obj.set_flags(None)
        obj.set_inlet_profile(prof, None, None, **kw)
        obj.set_macros(None, np.full((nz, ny, nx), 0.05), None, None, **kw)
    o.set_step(123456)
    sim.set_step(123456)
    o.set_inflow_turbulence(modes, 0.005, 0.5)
    sim.set_inflow_turbulence(modes, 0.005, 0.5)
    o.step(5)
    sim.step(5)
    g = [a.cpu().numpy().astype(np.float64) for a in sim.get_macros()]
    r = o.get_macros()
    for a, b in zip(g, r):
        assert np.abs(a[:, :, 0] - b[:, :, 0]).max() < 2e-7      # the inflow cells themselves
    assert max_err(sim, o) <= TOL32
    sim.close()


def test_set_inflow_turbulence_argument_errors(B):
    sim = B.Lbm(8, 8, 8, 1e-2, 0.1, 0.0, (0, 0, 0), (3, 4, 0, 0, 1, 2))
    m = np.zeros((2, 9)); m[:, 0] = 0.5; m[:, 4] = 1.0; m[:, 8] = 0.1
    with pytest.raises(B.LbmError):
        sim.set_inflow_turbulence(m, 0.01, 0.5)            # flags not set
    sim.set_flags(None)
    sim.set_inlet_profile(np.full(8, 0.05))
    with pytest.raises(B.LbmError):
        sim.set_inflow_turbulence(m, 0.01, 0.0)            # k_e must be > 0
    with pytest.raises(B.LbmError):
        sim.set_inflow_turbulence(m, -1.0, 0.5)
    bad = m.copy(); bad[0, 8] = -0.1
    with pytest.raises(B.LbmError):
        sim.set_inflow_turbulence(bad, 0.01, 0.5)
    with pytest.raises(B.LbmError):
        sim.set_inflow_turbulence(np.zeros((2000, 9)), 0.01, 0.5)
    sim.set_inflow_turbulence(None)                        # off while off: no-op
    sim.set_inflow_turbulence(m, 0.01, 0.5)
    sim.step(3)
    sim.set_flags(None)                                    # re-voxelising switches the fluctuations off
    sim.set_inlet_profile(np.full(8, 0.05))
    sim.close()


@pytest.mark.parametrize("fp64", [False, True])
def test_open_boundary_stack_together_matches_the_oracle(B, fp64):
    """Everything PAPER.md:175 / Table 1 PAPER.md:86 lists for the open faces at once: equilibrium velocity faces, global
    flux correction, sponge + buffer nudging, synthetic fluctuations on the active inflow cells (the DAMP + TURB
    instantiation of the step kernel), with the time mean accumulating."""
    from oracle import Oracle
    from paper_2607_04516_b200 import workloads as W
    nx, ny, nz = 44, 38, 20
    hm = np.zeros((ny, nx), dtype=np.int32)
    hm[14:20, 16:22] = 9
    hm[24:27, 28:33] = 5
    prof = (0.05 * np.log((np.arange(nz) + 0.5) / 0.1) / np.log(nz / 0.1)).clip(0)
    args = (nx, ny, nz, 2e-3, 0.1, 2e-4, (0.0, 0.0, 0.0), (3, 3, 3, 3, 1, 3))   # four lateral faces + top: all open
    target = np.stack([prof, 0.3 * prof, np.zeros(nz)])
    modes = W.inflow_modes(48, 41, 2 * np.pi / 30, np.pi, convect=(0.05, 0.015, 0.0))
    ux0 = np.broadcast_to(prof[:, None, None], (nz, ny, nx)).copy()
    o = Oracle(*args)
    sim = B.Lbm(*args, fp64=fp64)
    for obj, kw in ((o, {}), (sim, {"f64": True})):
        obj.set_flags(hm)
        obj.set_inlet_profile(prof, 0.3 * prof, None, **kw)
        obj.set_macros(None, ux0, 0.3 * ux0, None, **kw)
        b, a = obj.balance_flux()
        assert abs(a) < (1e-9 if (obj is o or fp64) else 2e-4)
        obj.set_damping((5, 8, 5, 5, 0, 6), (0.05, 0.15, 0.05, 0.05, 0.0, 0.2), target)
        obj.set_inflow_turbulence(modes, 0.003, 2 * np.pi / 12, 2.5)
        obj.mean_config(20, 5)
    o.step(100)
    sim.step(100)
    tol = TOL64 if fp64 else TOL32
    e = max_err(sim, o, f64=fp64)
    assert e <= tol, (fp64, e)
    gm, om = sim.get_mean(f64=fp64), o.get_mean()
    assert gm[3] == om[3] == 17
    em = max(float(np.abs(a.cpu().numpy().astype(np.float64) - b).max()) for a, b in zip(gm[:3], om[:3]))
    assert em <= tol, (fp64, em)
    sim.close()


# ---------------------------------------------------------------------------------------------- mesh voxeliser / solid masks

def _mesh_cases(W):
    rng = np.random.default_rng(5)
    boxes = []
    for _ in range(12):
        lo = rng.uniform(-3, 30, 3)
        boxes.append(W.box_mesh(lo, lo + rng.uniform(0.2, 14, 3)))
    yield "random overlapping boxes (generic coordinates)", np.concatenate(boxes), (37, 29, 23)
    yield "boxes with faces, edges and vertices on cell centres", np.concatenate(
        [W.box_mesh((1.5, 2.5, 1.5), (6.5, 5.5, 4.5)), W.box_mesh((6.5, 2.5, 1.5), (9.5, 7.5, 3.5)), W.box_mesh((12, 3, 0), (15, 6, 5))]), (20, 11, 8)
    yield "icosphere", W.icosphere_mesh((16.3, 15.6, 12.8), 10.7, 3), (33, 31, 27)
    yield "icosphere partly outside the box", W.icosphere_mesh((3.3, 28.6, 20.8), 9.2, 2), (33, 31, 27)
    sph = W.icosphere_mesh((10.2, 9.7, 8.1), 6.3, 2)
    yield "sphere with missing triangles (the vote repairs)", np.delete(sph, [3, 50, 121, 200], axis=0), (21, 20, 18)
    yield "slab on two legs (overhang)", np.concatenate(
        [W.box_mesh((5.2, 5.2, -1), (7.8, 9.8, 8.6)), W.box_mesh((15.2, 5.2, -1), (17.8, 9.8, 8.6)), W.box_mesh((5.2, 5.2, 6.4), (17.8, 9.8, 8.6))]), (24, 15, 12)
    yield "one huge triangle pair (ground sheet) + tiny slivers", np.concatenate(
        [W.box_mesh((-50, -50, -2), (200, 200, 1.3)), W.box_mesh((3.001, 3.001, 1.3), (3.9, 3.02, 5.7))]), (64, 40, 6)


@pytest.mark.parametrize("min_votes", [1, 2, 3])
def test_mesh_voxeliser_bit_exact_against_the_oracle(B, min_votes):
    """ray casting through grid columns, odd-even parity, three ray directions corroborated.  Flags and link
    words bit-exact on generic, degenerate, curved, clipped, leaky and overhanging meshes; host and device triangle arrays."""
    import torch
    from oracle import Oracle, mesh_voxel
    from paper_2607_04516_b200 import workloads as W
    faces = (3, 4, 2, 2, 1, 2)
    for name, tri, (nx, ny, nz) in _mesh_cases(W):
        mask = mesh_voxel.voxelise(tri, nx, ny, nz, min_votes)
        assert 0 < mask.sum() < mask.size, name
        o = Oracle(nx, ny, nz, 1e-3, 0.1, 0.0, (0, 0, 0), faces)
        o.set_flags_mask(None, mask)
        sim = B.Lbm(nx, ny, nz, 1e-3, 0.1, 0.0, (0, 0, 0), faces)
        sim.set_flags_mesh(tri, None, min_votes)
        check_flags_links(sim, o)
        sim.set_flags_mesh(torch.from_numpy(np.ascontiguousarray(tri, dtype=np.float32)).cuda(), None, min_votes)
        check_flags_links(sim, o)
        sim.close()


def test_mesh_on_terrain_heightmap_and_user_mask(B):
    """PAPER.md:51 Boolean merge: base + terrain as a heightmap, buildings as a mesh; and the same through a user mask
    (host and device).  An extruded-footprint city mesh reproduces the heightmap voxeliser exactly."""
    import torch
    from oracle import Oracle, mesh_voxel
    from paper_2607_04516_b200 import workloads as W
    nx, ny, nz = 70, 45, 20
    faces = (3, 4, 2, 2, 1, 2)
    hm = np.minimum(W.urban_heightmap(nx, ny, seed=9), nz - 4).astype(np.int32)
    terrain = (1 + np.arange(nx)[None, :] // 16 + 0 * np.arange(ny)[:, None]).astype(np.int32)
    tri = W.urban_mesh(hm)
    mask = mesh_voxel.voxelise(tri, nx, ny, nz)
    o = Oracle(nx, ny, nz, 1e-3, 0.1, 0.0, (0, 0, 0), faces)
    o.set_flags(np.maximum(hm, terrain))
    sim = B.Lbm(nx, ny, nz, 1e-3, 0.1, 0.0, (0, 0, 0), faces)
    sim.set_flags_mesh(tri, terrain)
    check_flags_links(sim, o)
    sim.set_flags_mask(terrain, mask)
    check_flags_links(sim, o)
    sim.set_flags_mask(torch.from_numpy(terrain).cuda(), torch.from_numpy(mask).cuda())
    check_flags_links(sim, o)
    sim.set_flags_mesh(None, terrain)                      # no triangles: the heightmap alone
    o.set_flags(terrain)
    check_flags_links(sim, o)
    with pytest.raises(B.LbmError):
        sim.set_flags_mesh(tri, None, 4)
    with pytest.raises(B.LbmError):
        sim.set_flags_mesh(W.box_mesh((0, 0, 0), (3000, 2, 2)), None)
    bad = tri.copy(); bad[0, 0, 0] = np.nan
    with pytest.raises(B.LbmError):
        sim.set_flags_mesh(bad, None)
    sim.set_flags_mesh(tri, terrain)                       # the handle is usable after an error
    o.set_flags(np.maximum(hm, terrain))
    check_flags_links(sim, o)
    sim.close()


@pytest.mark.parametrize("inplace", [False, True])
@pytest.mark.parametrize("fp64", [False, True])
def test_flow_around_mesh_voxelised_overhangs_matches_the_oracle(B, fp64, inplace):
    """Solids that no heightmap can express (a slab on two legs, a floating sphere): the step kernel works from the flags
    alone — bounce-back from below and above, sector completion inside hollow rows; 100 steps against the oracle.
    inplace: the same on one population buffer (wall links in all 18 directions through the link slots)."""
    from oracle import Oracle, mesh_voxel
    from paper_2607_04516_b200 import workloads as W
    nx, ny, nz = 56, 36, 24
    tri = np.concatenate([W.box_mesh((12.2, 8.2, -1), (14.8, 27.8, 12.6)), W.box_mesh((26.2, 8.2, -1), (28.8, 27.8, 12.6)),
                          W.box_mesh((12.2, 8.2, 9.4), (28.8, 27.8, 12.6)), W.icosphere_mesh((40.3, 18.1, 13.2), 5.4, 2)])
    hm = np.zeros((ny, nx), dtype=np.int32); hm[:, 33:36] = 2
    prof = (0.05 * np.log((np.arange(nz) + 0.5) / 0.1) / np.log(nz / 0.1)).clip(0)
    args = (nx, ny, nz, 2e-3, 0.1, 1e-4, (0, 0, 0), (3, 4, 2, 2, 1, 2))
    o = Oracle(*args)
    o.set_flags_mask(hm, mesh_voxel.voxelise(tri, nx, ny, nz))
    sim = B.Lbm(*args, fp64=fp64, inplace=inplace)
    sim.set_flags_mesh(tri, hm)
    check_flags_links(sim, o)
    fl = o.get_flags()
    assert fl[5, 18, 20] == 0 and fl[10, 18, 20] == 1 and fl[13, 18, 40] == 1 and fl[3, 18, 40] == 0
    ux0 = np.broadcast_to(prof[:, None, None], (nz, ny, nx)).copy()
    for obj, kw in ((o, {}), (sim, {"f64": True})):
        obj.set_inlet_profile(prof, None, None, **kw)
        obj.set_macros(None, ux0, None, None, **kw)
    o.step(101)
    sim.step(101)
    e = max_err(sim, o, f64=fp64)
    assert e <= (TOL64 if fp64 else TOL32), (fp64, inplace, e)
    sim.close()


def test_cooperative_multi_step_launch_equals_single_launches_bit_for_bit(B):
    """lbm_step(n) on a lattice whose grid is resident runs in one cooperative launch (step_loop_kernel); stepping one at a
    time uses one launch per step.  Same step body, same arithmetic: the states must be identical, with buildings,
    every face rule, damping zones, and a time mean whose sampling steps cut the run into several loops."""
    from paper_2607_04516_b200 import workloads as W
    wl = W.config1()
    prof = wl.inlet_profile[0].astype(np.float64)
    target = np.stack([prof, np.zeros_like(prof), np.zeros_like(prof)])
    sims = [B.from_workload(wl), B.from_workload(wl)]
    for s in sims:
        s.set_damping((0, 6, 0, 0, 0, 5), (0, 0.1, 0, 0, 0, 0.2), target)
        s.mean_config(10, 7)
    l0 = [s.launch_count() for s in sims]
    sims[0].step(101)
    for _ in range(101):
        sims[1].step(1)
    n_loop, n_single = sims[0].launch_count() - l0[0], sims[1].launch_count() - l0[1]
    assert n_single == 101 and n_loop < 40, (n_loop, n_single)
    assert np.array_equal(sims[0].get_state(out="host"), sims[1].get_state(out="host"))
    m0, m1 = sims[0].get_mean(out="host"), sims[1].get_mean(out="host")
    assert m0[3] == m1[3] == 14
    for a, b in zip(m0[:3], m1[:3]):
        assert np.array_equal(a, b)
    for s in sims:
        s.close()

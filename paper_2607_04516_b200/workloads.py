"""Seeded synthetic inputs for the five BASELINE.json configs (and their crops).

This module holds NO arithmetic of the method — no lattice table, no
equilibrium, no collision.  It only produces the arrays a caller hands to the
solver (heightmaps, boundary wind profiles, initial macroscopic fields) and the
scalar parameters of each config, so that the CUDA library and the CPU oracle
can be fed bit-identical inputs.  numpy only.

The arrays stand in for the paper's datasets (3D-GloBFP buildings and NASADEM
terrain; Guangzhou lidar profiles), none of
which exist on this box; shapes follow the paper's workload (5 m cells,
kilometre-scale; building short sides mostly < 50 m = 10
cells).  Recipes: DESIGN.md "Input recipe" (= SURVEY.md §8(d)).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

# face types of the C ABI (include/lbm.h), order x-,x+,y-,y+,z-,z+
PERIODIC, WALL, FREE_SLIP, EQ_FIXED, EQ_OUTFLOW = 0, 1, 2, 3, 4


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    nu0: float
    Cs: float
    f_cor: float
    F: tuple
    faces: tuple
    steps: int
    height: np.ndarray                      # int32 [ny][nx]
    inlet_profile: tuple | None = None      # (u[nz], v[nz] | None, w[nz] | None) float32
    init: tuple | None = None               # (rho, ux, uy, uz) float32 [nz][ny][nx], entries may be None
    mean_start: int = 0
    mean_every: int = 0
    extra: dict = field(default_factory=dict)

    @property
    def cells(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)


# --------------------------------------------------------------------------- profiles

def log_law_profile(nz: int, u_ref: float, zeta_ref: float, z0: float) -> np.ndarray:
    """|U|(zeta) = u_ref ln(zeta/z0)/ln(zeta_ref/z0) at cell centres zeta = z + 1/2, clipped at >= 0."""
    zeta = np.arange(nz, dtype=np.float64) + 0.5
    u = u_ref * np.log(zeta / z0) / math.log(zeta_ref / z0)
    return np.maximum(u, 0.0).astype(np.float32)


def veering_profile(nz: int, u_ref: float, zeta_ref: float, z0: float, seed: int,
                    theta_max_deg: float = 60.0, jitter: float = 0.1):
    """Config-4 inlet: log-law speed, direction turning 0..theta_max over the depth with a
    seeded +-10 % perturbation  theta(zeta) = theta_max (zeta/nz) (1 + jitter s(zeta)),
    s = sum of 3 seeded sine modes normalised to max|s| = 1."""
    rng = np.random.Generator(np.random.PCG64(seed))
    zeta = np.arange(nz, dtype=np.float64) + 0.5
    amp = rng.uniform(0.5, 1.0, size=3)
    phase = rng.uniform(0.0, 2.0 * math.pi, size=3)
    s = sum(a * np.sin(2.0 * math.pi * (m + 1) * zeta / nz + p) for m, (a, p) in enumerate(zip(amp, phase)))
    s = s / np.max(np.abs(s))
    theta = np.deg2rad(theta_max_deg) * (zeta / nz) * (1.0 + jitter * s)
    speed = log_law_profile(nz, u_ref, zeta_ref, z0).astype(np.float64)
    return (speed * np.cos(theta)).astype(np.float32), (speed * np.sin(theta)).astype(np.float32)


def inflow_modes(n: int, seed: int, k_min: float, k_max: float, convect=(0.0, 0.0, 0.0)) -> np.ndarray:
    """The random draws of the synthetic inflow fluctuations (Table 1), as an input table
    [n][9] = kappa[3], sigma[3], psi, omega, dkappa — no spectrum, no amplitudes: those are the method's arithmetic
    and live in the library / the oracle.  Wavenumber magnitudes are n equal shells between k_min and k_max (shell
    centres, dkappa = the shell width); directions are uniform on the sphere (phi ~ U(0, 2 pi), cos(theta) ~ U(-1, 1));
    sigma is a unit vector in the plane normal to kappa at a uniform angle; psi ~ U(0, 2 pi); omega = kappa . convect
    (frozen turbulence carried with the velocity `convect`, lattice units)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    dk = (k_max - k_min) / n
    kmag = k_min + (np.arange(n) + 0.5) * dk
    phi = rng.uniform(0.0, 2.0 * math.pi, n)
    ct = rng.uniform(-1.0, 1.0, n)
    st = np.sqrt(1.0 - ct * ct)
    e = np.stack([st * np.cos(phi), st * np.sin(phi), ct], axis=1)                  # unit wave-vector directions
    a = np.stack([-np.sin(phi), np.cos(phi), np.zeros(n)], axis=1)                  # two unit vectors spanning the normal plane
    b = np.cross(e, a)
    al = rng.uniform(0.0, 2.0 * math.pi, n)
    sig = np.cos(al)[:, None] * a + np.sin(al)[:, None] * b
    psi = rng.uniform(0.0, 2.0 * math.pi, n)
    kap = kmag[:, None] * e
    om = kap @ np.asarray(convect, dtype=np.float64)
    return np.concatenate([kap, sig, psi[:, None], om[:, None], np.full((n, 1), dk)], axis=1)


# --------------------------------------------------------------------------- heightmaps

def block_heightmap(nx, ny, x0, x1, y0, y1, h) -> np.ndarray:
    hm = np.zeros((ny, nx), dtype=np.int32)
    hm[y0:y1 + 1, x0:x1 + 1] = h
    return hm


def urban_heightmap(nx: int, ny: int, seed: int, plan_fraction: float = 0.35, wmin: int = 2, wmax: int = 12,
                    h_median: float = 6.0, h_sigma: float = 0.6, h_max: int = 40, x_margin: int = 8) -> np.ndarray:
    """Rectangular footprints w,l ~ U{wmin..wmax}, height = clip(round(h_median exp(sigma N(0,1))), 1, h_max),
    uniform positions with a building-free margin at the x faces, overlaps resolved by max, drawn until the
    built plan-area fraction (of the whole map) reaches plan_fraction."""
    rng = np.random.Generator(np.random.PCG64(seed))
    hm = np.zeros((ny, nx), dtype=np.int32)
    target = plan_fraction * nx * ny
    built = 0
    batch = 256
    while built < target:
        w = rng.integers(wmin, wmax + 1, size=batch)
        l = rng.integers(wmin, wmax + 1, size=batch)
        h = np.clip(np.rint(h_median * np.exp(h_sigma * rng.standard_normal(batch))), 1, h_max).astype(np.int32)
        ux = rng.random(batch)
        uy = rng.random(batch)
        for k in range(batch):
            xs = x_margin + int(ux[k] * (nx - 2 * x_margin - w[k] + 1))
            ys = int(uy[k] * (ny - l[k] + 1))
            blk = hm[ys:ys + l[k], xs:xs + w[k]]
            built += int(np.count_nonzero(blk == 0))
            np.maximum(blk, h[k], out=blk)
            if built >= target:
                break
    return hm


# --------------------------------------------------------------------------- configs

def config1() -> Workload:
    """Tiny block flow, 64x32x32 (BASELINE.json configs[0])."""
    nx, ny, nz = 64, 32, 32
    hm = block_heightmap(nx, ny, 16, 23, 12, 19, 16)
    u = log_law_profile(nz, 0.05, 16.0, 0.1)
    ux = np.broadcast_to(u[:, None, None], (nz, ny, nx)).astype(np.float32).copy()
    return Workload("C1_block_64x32x32", nx, ny, nz, 1e-3, 0.1, 1e-3, (0.0, 0.0, 0.0),
                    (EQ_FIXED, EQ_OUTFLOW, PERIODIC, PERIODIC, WALL, FREE_SLIP), 200, hm,
                    inlet_profile=(u, None, None), init=(None, ux, None, None))


def config2(Cs: float = 0.0, n: int = 128, nz: int | None = None) -> Workload:
    """Periodic Taylor-Green + Coriolis, n^3 (BASELINE.json configs[1]); run A Cs=0, run B Cs=0.1."""
    nz = n if nz is None else nz
    k = 2.0 * math.pi / n
    u0, ub = 0.04, 0.02
    x = np.arange(n, dtype=np.float64)
    X, Y = np.meshgrid(x, x, indexing="xy")  # [y][x]
    ux2 = u0 * np.sin(k * X) * np.cos(k * Y) + ub
    uy2 = -u0 * np.cos(k * X) * np.sin(k * Y)
    rho2 = 1.0 - 0.75 * u0 * u0 * (np.cos(2 * k * X) + np.cos(2 * k * Y))
    ext = lambda a: np.broadcast_to(a[None], (nz, n, n)).astype(np.float32).copy()  # noqa: E731
    return Workload(f"C2_tgv_{n}x{n}x{nz}_Cs{Cs:g}", n, n, nz, 2e-3, Cs, 2e-4, (0.0, 0.0, 0.0),
                    (PERIODIC,) * 6, 1000, np.zeros((n, n), dtype=np.int32),
                    init=(ext(rho2), ext(ux2), ext(uy2), None), extra={"k": k, "u0": u0, "ub": ub})


def _urban(name, nx, ny, nz, hm, u_ref, zeta_ref, z0, nu0, f_cor, steps, faces=None) -> Workload:
    u = log_law_profile(nz, u_ref, zeta_ref, z0)
    ux = np.broadcast_to(u[:, None, None], (nz, ny, nx)).astype(np.float32).copy()
    faces = faces or (EQ_FIXED, EQ_OUTFLOW, FREE_SLIP, FREE_SLIP, WALL, FREE_SLIP)
    return Workload(name, nx, ny, nz, nu0, 0.1, f_cor, (0.0, 0.0, 0.0), faces, steps, hm,
                    inlet_profile=(u, None, None), init=(None, ux, None, None),
                    mean_start=steps // 2, mean_every=10)


def config3(nx: int = 400, ny: int = 400, nz: int = 100) -> Workload:
    """Synthetic 2 km urban domain at 5 m, 400x400x100 (BASELINE.json configs[2]); crops keep the recipe."""
    hm = urban_heightmap(400, 400, seed=3)[:ny, :nx].copy()
    return _urban(f"C3_urban_{nx}x{ny}x{nz}", nx, ny, nz, hm, 0.08, 20.0, 0.2, 1e-4, 2.9e-6, 20000)


def config4(nx: int = 800, ny: int = 800, nz: int = 200) -> Workload:
    """Refined urban domain at 2.5 m, 800x800x200 (BASELINE.json configs[3]): config-3 map x2 in cells,
    heights x2; veering inlet on x-, y-, y+; outflow on x+."""
    hm = np.kron(urban_heightmap(400, 400, seed=3), np.ones((2, 2), dtype=np.int32)).astype(np.int32) * 2
    hm = hm[:ny, :nx].copy()
    u, v = veering_profile(nz, 0.08, 40.0, 0.4, seed=4)
    bc = lambda a: np.broadcast_to(a[:, None, None], (nz, ny, nx)).astype(np.float32).copy()  # noqa: E731
    return Workload(f"C4_urban_{nx}x{ny}x{nz}", nx, ny, nz, 5e-5, 0.1, 1.5e-6, (0.0, 0.0, 0.0),
                    (EQ_FIXED, EQ_OUTFLOW, EQ_FIXED, EQ_FIXED, WALL, FREE_SLIP), 20000, hm,
                    inlet_profile=(u, v, None), init=(None, bc(u), bc(v), None), mean_start=10000, mean_every=10)


def config5_precursor(nx: int = 256, ny: int = 256, nz: int = 200) -> Workload:
    """Periodic precursor box 256x256x200 (BASELINE.json configs[4], first half): flat ground, pressure-gradient
    force 1e-6 + Coriolis, initial log-law + 2 % seeded noise."""
    rng = np.random.Generator(np.random.PCG64(55))
    u = log_law_profile(nz, 0.08, 20.0, 0.2)
    base = np.broadcast_to(u[:, None, None], (nz, ny, nx)).astype(np.float64)
    noise = lambda: (0.02 * 0.08 * rng.standard_normal((nz, ny, nx)))  # noqa: E731
    ux = (base + noise()).astype(np.float32)
    uy = noise().astype(np.float32)
    uz = noise().astype(np.float32)
    return Workload(f"C5_precursor_{nx}x{ny}x{nz}", nx, ny, nz, 1e-4, 0.1, 2.9e-6, (1e-6, 0.0, 0.0),
                    (PERIODIC, PERIODIC, PERIODIC, PERIODIC, WALL, FREE_SLIP), 10000,
                    np.zeros((ny, nx), dtype=np.int32), init=(None, ux, uy, uz), extra={"sample_plane_x": nx // 2})


def config5_main(nx: int = 1200, ny: int = 1200, nz: int = 200) -> Workload:
    """Main urban domain 1200x1200x200 of config 5 (seed-5 heightmap with config-3 statistics); its x- inlet is
    fed every step from the precursor plane."""
    hm = urban_heightmap(1200, 1200, seed=5)[:ny, :nx].copy()
    return _urban(f"C5_main_{nx}x{ny}x{nz}", nx, ny, nz, hm, 0.08, 20.0, 0.2, 1e-4, 2.9e-6, 10000)


def mean_profile(u: np.ndarray, flags: np.ndarray, solid_code: int = 1) -> np.ndarray:
    """Horizontal average over non-SOLID cells of each level z (post-processing, not part of the method)."""
    fluid = flags != solid_code
    cnt = np.maximum(fluid.sum(axis=(1, 2)), 1)
    return (np.where(fluid, u, 0.0).sum(axis=(1, 2), dtype=np.float64)) / cnt


# --------------------------------------------------------------------------- triangle meshes (inputs of the mesh voxeliser)

def box_mesh(lo, hi) -> np.ndarray:
    """12 outward-oriented triangles of the axis-aligned box [lo, hi]; float32 [12][3][3], lattice units."""
    x0, y0, z0 = lo
    x1, y1, z1 = hi
    c = np.array([[x0, y0, z0], [x1, y0, z0], [x1, y1, z0], [x0, y1, z0],
                  [x0, y0, z1], [x1, y0, z1], [x1, y1, z1], [x0, y1, z1]], dtype=np.float64)
    quads = [(0, 3, 2, 1), (4, 5, 6, 7), (0, 1, 5, 4), (2, 3, 7, 6), (1, 2, 6, 5), (3, 0, 4, 7)]
    tri = []
    for a, b, d, e in quads:
        tri.append([c[a], c[b], c[d]])
        tri.append([c[a], c[d], c[e]])
    return np.asarray(tri, dtype=np.float32)


def icosphere_mesh(centre, radius: float, subdivisions: int = 2) -> np.ndarray:
    """Closed triangle mesh inscribed in a sphere (icosahedron subdivided); float32 [20 * 4^s][3][3]."""
    t = (1.0 + math.sqrt(5.0)) / 2.0
    v = [(-1, t, 0), (1, t, 0), (-1, -t, 0), (1, -t, 0), (0, -1, t), (0, 1, t), (0, -1, -t), (0, 1, -t),
         (t, 0, -1), (t, 0, 1), (-t, 0, -1), (-t, 0, 1)]
    v = [np.asarray(p, dtype=np.float64) / math.sqrt(1 + t * t) for p in v]
    f = [(0, 11, 5), (0, 5, 1), (0, 1, 7), (0, 7, 10), (0, 10, 11), (1, 5, 9), (5, 11, 4), (11, 10, 2), (10, 7, 6), (7, 1, 8),
         (3, 9, 4), (3, 4, 2), (3, 2, 6), (3, 6, 8), (3, 8, 9), (4, 9, 5), (2, 4, 11), (6, 2, 10), (8, 6, 7), (9, 8, 1)]
    tri = [[v[a], v[b], v[c]] for a, b, c in f]
    for _ in range(subdivisions):
        nxt = []
        for a, b, c in tri:
            ab, bc, ca = [(p + q) / np.linalg.norm(p + q) for p, q in ((a, b), (b, c), (c, a))]
            nxt += [[a, ab, ca], [b, bc, ab], [c, ca, bc], [ab, bc, ca]]
        tri = nxt
    return (np.asarray(tri) * radius + np.asarray(centre, dtype=np.float64)).astype(np.float32)


def urban_mesh(height: np.ndarray, z_shift: float = 0.0) -> np.ndarray:
    """One closed box per maximal run of equal non-zero height along x in every row of a heightmap (buildings as
    extruded footprints, the way a city model delivers them); float32 [n][3][3]."""
    ny, nx = height.shape
    out = []
    for y in range(ny):
        x = 0
        while x < nx:
            h = int(height[y, x])
            x1 = x
            while x1 < nx and int(height[y, x1]) == h:
                x1 += 1
            if h > 0:
                out.append(box_mesh((x, y, -1.0 + z_shift), (x1, y + 1, h + z_shift)))
            x = x1
    return np.concatenate(out) if out else np.zeros((0, 3, 3), dtype=np.float32)


def density_current(nx: int = 256, nz: int = 64, ny: int = 2, d_theta: float = -15.0, theta_ref: float = 300.0):
    """Synthetic stand-in for the density-current workload ("initially quiescent, neutrally stratified
    atmosphere with a cold elliptical potential-temperature perturbation in a 25.6 km by 6.4 km domain"): a 4:1 x-z box,
    thin and periodic in y, at rest; theta = theta_ref + d_theta (cos(pi L) + 1) / 2 inside the ellipse L <= 1 centred on
    the domain's vertical mid-plane at 3/6.4 of the height, radii 4/25.6 of the length and 2/6.4 of the height.
    Returns (faces, theta[nz][ny][nx] float64).  Input generation only: no arithmetic of the method."""
    x = (np.arange(nx) + 0.5) / nx          # fractions of the 25.6 km length
    z = (np.arange(nz) + 0.5) / nz          # fractions of the 6.4 km height
    Lx = (x - 0.5) / (4.0 / 25.6)
    Lz = (z - 3.0 / 6.4) / (2.0 / 6.4)
    L = np.sqrt(Lx[None, :] ** 2 + Lz[:, None] ** 2)
    pert = np.where(L <= 1.0, 0.5 * d_theta * (np.cos(np.pi * L) + 1.0), 0.0)
    theta = theta_ref + np.repeat(pert[:, None, :], ny, axis=1)
    faces = (FREE_SLIP, FREE_SLIP, PERIODIC, PERIODIC, WALL, FREE_SLIP)
    return faces, np.ascontiguousarray(theta, dtype=np.float64)


def thermal_city(nx: int = 400, ny: int = 400, nz: int = 100, seed: int = 7) -> Workload:
    """Timing / full-size parity workload of the thermal path: config 3's city in a CLOSED box (free-slip sides and top, WALL
    ground — the thermal lattice takes no open faces), at rest, theta = 300 + seeded N(0, 1) K, buoyancy on.
    extra["thermal"] = (alpha, g_beta, theta_ref); extra["theta"] = the initial field (float32)."""
    c3 = config3(nx, ny, nz)
    rng = np.random.Generator(np.random.PCG64(seed))
    theta = (300.0 + rng.standard_normal((nz, ny, nx))).astype(np.float32)
    return Workload("thermal_city", nx, ny, nz, c3.nu0, c3.Cs, c3.f_cor, (1e-6, 0.0, 0.0),
                    (FREE_SLIP, FREE_SLIP, FREE_SLIP, FREE_SLIP, WALL, FREE_SLIP), 1000, c3.height,
                    extra={"thermal": (1e-2, 1e-5, 300.0), "theta": theta})   # alpha 1e-2: tau_theta = 0.54 (at 1e-3 = 0.504 the
                    # cell-scale temperature noise, fed back through the buoyancy, blows the BGK thermal lattice up after ~500 steps)


def density_current_benchmark(dx_m: float = 100.0, u_lat: float = 0.1):
    """The density-current benchmark of PAPER.md:121-125 in lattice units (input generation and unit conversion only).

    Physical set-up as the paper describes it: quiescent neutral atmosphere, 25.6 km x 6.4 km (x >= 0 half of the symmetric
    problem: the x- face is the symmetry plane), cold elliptical perturbation theta' = -15 (cos(pi L) + 1) / 2 K for L <= 1
    centred at (0, 3 km) with radii (4 km, 2 km), constant kinematic viscosity and diffusivity 75 m^2/s (the "AV75"
    configuration), g = 9.81 m/s^2, theta_0 = 300 K, free-slip box.  Lattice scaling: dx = dx_m, dt chosen so that 35 m/s
    (the flow's peak speed) maps to u_lat.  The thermal lattice carries the PERTURBATION (theta_ref = 0): it transports theta
    conservatively, so an absolute 300 K would turn the O(1e-3) density waves of the weakly compressible flow into O(1 K) noise.
    Returns dict(nx, ny, nz, faces, nu, alpha, g_beta, theta_ref, theta[nz][1][nx] float64, dt, dx, x_m[nx])."""
    nx, nz = int(round(25600.0 / dx_m)), int(round(6400.0 / dx_m))
    dt = dx_m * u_lat / 35.0
    nu = 75.0 * dt / dx_m ** 2
    g_beta = 9.81 / 300.0 * dt * dt / dx_m
    x = (np.arange(nx) + 0.5) * dx_m
    z = (np.arange(nz) + 0.5) * dx_m
    L = np.sqrt((x[None, :] / 4000.0) ** 2 + ((z[:, None] - 3000.0) / 2000.0) ** 2)
    pert = np.where(L <= 1.0, -7.5 * (np.cos(np.pi * L) + 1.0), 0.0)
    return dict(nx=nx, ny=1, nz=nz, faces=(FREE_SLIP, FREE_SLIP, PERIODIC, PERIODIC, FREE_SLIP, FREE_SLIP), nu=nu, alpha=nu,
                g_beta=g_beta, theta_ref=0.0, theta=np.ascontiguousarray(pert[:, None, :]), dt=dt, dx=dx_m, x_m=x)


def front_position_km(theta_pert: np.ndarray, x_m: np.ndarray, level: float = -1.0) -> float:
    """Front of a cold pool: the largest x where min_z theta' crosses `level` (linear interpolation between columns).
    theta_pert is [nz][nx].  A diagnostic on outputs (no arithmetic of the method)."""
    prof = np.asarray(theta_pert, dtype=np.float64).min(axis=0)
    cols = np.where(prof <= level)[0]
    if cols.size == 0:
        return float("nan")
    i = int(cols.max())
    xf = x_m[i]
    if i + 1 < len(x_m) and prof[i + 1] > level:
        xf = x_m[i] + (x_m[i + 1] - x_m[i]) * (prof[i] - level) / (prof[i] - prof[i + 1])
    return float(xf) / 1000.0

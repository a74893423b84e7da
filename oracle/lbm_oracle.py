"""ctypes binding of oracle/lbm_oracle.c (TEST INFRASTRUCTURE — see that file's header).

``build()`` compiles the C file with gcc (``-O3 -fopenmp``, no fast-math) into
``oracle/liblbm_oracle.so``; everything else is argument marshalling.
Arrays are numpy float64, C order ``[z][y][x]``.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lbm_oracle.c")
_SO = os.path.join(_HERE, "liblbm_oracle.so")
_lib = None

FLUID, SOLID, EQ_FIXED, EQ_OUTFLOW = 0, 1, 2, 3
PERIODIC, WALL, FREE_SLIP, FACE_EQ_FIXED, FACE_EQ_OUTFLOW = 0, 1, 2, 3, 4


def build(force: bool = False) -> str:
    """Compile the oracle if the .so is missing or older than the source."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O3", "-fopenmp", "-std=c99", "-shared", "-fPIC", "-o", _SO, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    lib = C.CDLL(_SO)
    dp = C.POINTER(C.c_double)
    lib.oracle_create.restype = C.c_void_p
    lib.oracle_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, dp]
    lib.oracle_destroy.restype = None
    lib.oracle_destroy.argtypes = [C.c_void_p]
    lib.oracle_get_step.restype = C.c_long
    lib.oracle_get_step.argtypes = [C.c_void_p]
    lib.oracle_set_step.argtypes = [C.c_void_p, C.c_long]
    lib.oracle_mean_config.argtypes = [C.c_void_p, C.c_long, C.c_int]
    for name in ("oracle_set_boundaries", "oracle_set_flags", "oracle_get_flags", "oracle_get_links",
                 "oracle_set_inlet_profile", "oracle_set_inlet_plane", "oracle_set_macros", "oracle_step",
                 "oracle_get_macros", "oracle_mean_reset", "oracle_get_mean",
                 "oracle_get_state", "oracle_set_state", "oracle_lattice", "oracle_feq", "oracle_collide_cell",
                 "oracle_collide_cell_vec", "oracle_set_coriolis", "oracle_balance_flux",
                 "oracle_collide_cell_damped", "oracle_set_damping", "oracle_get_damping",
                 "oracle_vk_spectrum", "oracle_set_inflow_turbulence", "oracle_set_flags_mask",
                 "oracle_set_theta", "oracle_get_theta", "oracle_get_thermal_state", "oracle_heq", "oracle_round_half", "oracle_set_storage16", "oracle_set_thermal_walls", "oracle_set_inlet_theta"):
        getattr(lib, name).restype = C.c_int
    lib.oracle_set_thermal.restype = C.c_int
    lib.oracle_set_thermal.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double]
    lib.oracle_heq.argtypes = [C.c_double, dp, dp]
    _lib = lib
    return lib


def _d(a):
    """float64 C-contiguous view/copy and its pointer (None -> NULL)."""
    if a is None:
        return None, None
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def lattice():
    """(c[19,3] int, w[19] float64, opposite[19] int) as the oracle defines them."""
    lib = _load()
    c = np.zeros((19, 3), dtype=np.int32)
    w = np.zeros(19, dtype=np.float64)
    opp = np.zeros(19, dtype=np.int32)
    lib.oracle_lattice(c.ctypes.data_as(C.c_void_p), w.ctypes.data_as(C.c_void_p), opp.ctypes.data_as(C.c_void_p))
    return c, w, opp


def feq(rho, u):
    lib = _load()
    u, up = _d(np.asarray(u, dtype=np.float64))
    out = np.zeros(19)
    lib.oracle_feq(C.c_double(rho), up, out.ctypes.data_as(C.c_void_p))
    return out


def collide_cell(f, nu0, Cs, fcor, F):
    """One cell's step 4b-4e.  Returns (g[19], rho, u[3], tau)."""
    lib = _load()
    f, fp = _d(f)
    F, Fp = _d(np.asarray(F, dtype=np.float64))
    g = np.zeros(19)
    rho = C.c_double()
    u = np.zeros(3)
    tau = C.c_double()
    lib.oracle_collide_cell(fp, C.c_double(nu0), C.c_double(Cs), C.c_double(fcor), Fp,
                            g.ctypes.data_as(C.c_void_p), C.byref(rho), u.ctypes.data_as(C.c_void_p), C.byref(tau))
    return g, rho.value, u, tau.value


def collide_cell_vec(f, nu0, Cs, fvec, F):
    """One cell's step 4b-4e with the full Coriolis vector f = 2 Omega.  Returns (g[19], rho, u[3], tau)."""
    lib = _load()
    f, fp = _d(f)
    F, Fp = _d(np.asarray(F, dtype=np.float64))
    fv, fvp = _d(np.asarray(fvec, dtype=np.float64))
    g = np.zeros(19)
    rho = C.c_double()
    u = np.zeros(3)
    tau = C.c_double()
    lib.oracle_collide_cell_vec(fp, C.c_double(nu0), C.c_double(Cs), fvp, Fp,
                                g.ctypes.data_as(C.c_void_p), C.byref(rho), u.ctypes.data_as(C.c_void_p), C.byref(tau))
    return g, rho.value, u, tau.value


def collide_cell_damped(f, nu0, Cs, fvec, F, sigma, ut):
    """One cell's step 4b-4e inside a damping zone (coefficient sigma, target velocity ut).  Returns (g, rho, u, tau)."""
    lib = _load()
    f, fp = _d(f)
    F, Fp = _d(np.asarray(F, dtype=np.float64))
    fv, fvp = _d(np.asarray(fvec, dtype=np.float64))
    ut, utp = _d(np.asarray(ut, dtype=np.float64))
    g = np.zeros(19)
    rho = C.c_double()
    u = np.zeros(3)
    tau = C.c_double()
    lib.oracle_collide_cell_damped(fp, C.c_double(nu0), C.c_double(Cs), fvp, Fp, C.c_double(sigma), utp,
                                   g.ctypes.data_as(C.c_void_p), C.byref(rho), u.ctypes.data_as(C.c_void_p), C.byref(tau))
    return g, rho.value, u, tau.value


def heq(theta, u):
    """D3Q7 thermal equilibrium h_eq[7] (directions 0..6 of the lattice)."""
    lib = _load()
    u, up = _d(np.asarray(u, dtype=np.float64))
    out = np.zeros(7)
    lib.oracle_heq(float(theta), up, out.ctypes.data_as(C.POINTER(C.c_double)))
    return out


def round_half(x):
    """The oracle's round-to-binary16 (ties to even, subnormals kept) of each element; float64 in and out."""
    lib = _load()
    x, xp = _d(np.atleast_1d(x))
    out = np.zeros(x.size)
    lib.oracle_round_half(C.c_int(x.size), xp, out.ctypes.data_as(C.c_void_p))
    return out.reshape(x.shape)


def vk_spectrum(k, u_rms, k_e, k_eta=0.0):
    """von Karman-Pao energy spectrum E(k) (k_eta = 0: no Pao cut-off)."""
    lib = _load()
    k, kp = _d(np.atleast_1d(k))
    E = np.zeros(k.size)
    lib.oracle_vk_spectrum(C.c_int(k.size), kp, C.c_double(u_rms), C.c_double(k_e), C.c_double(k_eta),
                           E.ctypes.data_as(C.c_void_p))
    return E


class Oracle:
    """FP64 CPU LBM; same call names as the product binding, float64 arrays."""

    def __init__(self, nx, ny, nz, nu0, Cs=0.0, f_cor=0.0, F=(0.0, 0.0, 0.0), faces=None):
        self._lib = _load()
        F = np.atleast_1d(np.asarray(F, dtype=np.float64))
        if F.size == 1:
            F = np.array([F[0], 0.0, 0.0])
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.shape = (self.nz, self.ny, self.nx)
        self._h = self._lib.oracle_create(self.nx, self.ny, self.nz, C.c_double(nu0), C.c_double(Cs),
                                          C.c_double(f_cor), F.ctypes.data_as(C.POINTER(C.c_double)))
        if not self._h:
            raise MemoryError("oracle_create failed")
        if faces is not None:
            self.set_boundaries(faces)

    def close(self):
        if getattr(self, "_h", None):
            self._lib.oracle_destroy(C.c_void_p(self._h))
            self._h = None

    __del__ = close

    def _chk(self, rc, what):
        if rc != 0:
            raise RuntimeError(f"oracle {what} failed: {rc}")

    def set_storage16(self, on=True):
        """Every population written from now on is kept as binary16 of its shifted value."""
        self._chk(self._lib.oracle_set_storage16(C.c_void_p(self._h), int(bool(on))), "set_storage16")

    def set_coriolis(self, fvec):
        """Full Coriolis vector f = 2 Omega (lattice units); (0, 0, f_cor) is the scalar form."""
        a, ap = _d(np.asarray(fvec, dtype=np.float64).reshape(3))
        self._chk(self._lib.oracle_set_coriolis(C.c_void_p(self._h), ap), "set_coriolis")

    def set_damping(self, width, peak, target=None):
        """Sponge / buffer zones: per-face width (cells) and peak coefficient, target profile [3][nz]."""
        w = np.ascontiguousarray(width, dtype=np.int32).reshape(6)
        pk, pkp = _d(np.asarray(peak, dtype=np.float64).reshape(6))
        t, tp = (None, None) if target is None else _d(np.asarray(target, dtype=np.float64).reshape(3, self.nz))
        self._chk(self._lib.oracle_set_damping(C.c_void_p(self._h), w.ctypes.data_as(C.c_void_p), pkp, tp), "set_damping")

    def get_damping(self):
        s = np.zeros(self.shape)
        self._chk(self._lib.oracle_get_damping(C.c_void_p(self._h), s.ctypes.data_as(C.c_void_p)), "get_damping")
        return s

    def set_inflow_turbulence(self, modes, u_rms=0.0, k_e=1.0, k_eta=0.0):
        """Synthetic von Karman fluctuations on active inflow cells; modes [n][9] = kappa, sigma, psi, omega, dkappa
        (None / empty: off)."""
        if modes is None or len(modes) == 0:
            self._chk(self._lib.oracle_set_inflow_turbulence(C.c_void_p(self._h), 0, None, C.c_double(0), C.c_double(1),
                                                             C.c_double(0)), "set_inflow_turbulence")
            return
        m, mp = _d(np.asarray(modes, dtype=np.float64).reshape(-1, 9))
        self._chk(self._lib.oracle_set_inflow_turbulence(C.c_void_p(self._h), m.shape[0], mp, C.c_double(u_rms),
                                                         C.c_double(k_e), C.c_double(k_eta)), "set_inflow_turbulence")

    def balance_flux(self):
        """Global flux-balancing correction of the EQ_FIXED face velocities; returns (flux_before, flux_after)."""
        a, b = C.c_double(), C.c_double()
        self._chk(self._lib.oracle_balance_flux(C.c_void_p(self._h), C.byref(a), C.byref(b)), "balance_flux")
        return a.value, b.value

    def set_boundaries(self, faces):
        a = np.ascontiguousarray(faces, dtype=np.int32)
        assert a.shape == (6,)
        self._chk(self._lib.oracle_set_boundaries(C.c_void_p(self._h), a.ctypes.data_as(C.c_void_p)), "set_boundaries")

    def set_flags(self, height=None):
        if height is None:
            height = np.zeros((self.ny, self.nx), dtype=np.int32)
        a = np.ascontiguousarray(height, dtype=np.int32)
        assert a.shape == (self.ny, self.nx)
        self._chk(self._lib.oracle_set_flags(C.c_void_p(self._h), a.ctypes.data_as(C.c_void_p)), "set_flags")

    def set_flags_mask(self, height=None, solid=None):
        """Heightmap (or None) merged with a general solid mask uint8 [nz][ny][nx] (non-zero = SOLID)."""
        if height is None:
            height = np.zeros((self.ny, self.nx), dtype=np.int32)
        a = np.ascontiguousarray(height, dtype=np.int32)
        assert a.shape == (self.ny, self.nx)
        m = None
        if solid is not None:
            m = np.ascontiguousarray(solid, dtype=np.uint8)
            assert m.shape == self.shape
        self._chk(self._lib.oracle_set_flags_mask(C.c_void_p(self._h), a.ctypes.data_as(C.c_void_p),
                                                  m.ctypes.data_as(C.c_void_p) if m is not None else None), "set_flags_mask")

    def get_flags(self):
        out = np.zeros(self.shape, dtype=np.uint8)
        self._chk(self._lib.oracle_get_flags(C.c_void_p(self._h), out.ctypes.data_as(C.c_void_p)), "get_flags")
        return out

    def get_links(self):
        out = np.zeros(self.shape, dtype=np.uint32)
        self._chk(self._lib.oracle_get_links(C.c_void_p(self._h), out.ctypes.data_as(C.c_void_p)), "get_links")
        return out

    def set_inlet_profile(self, u, v=None, w=None):
        u, up = _d(u)
        v, vp = _d(v)
        w, wp = _d(w)
        assert u.shape == (self.nz,)
        self._chk(self._lib.oracle_set_inlet_profile(C.c_void_p(self._h), up, vp, wp), "set_inlet_profile")

    def set_inlet_plane(self, face, uvw):
        uvw, p = _d(uvw)
        self._chk(self._lib.oracle_set_inlet_plane(C.c_void_p(self._h), int(face), p), "set_inlet_plane")

    def set_macros(self, rho=None, ux=None, uy=None, uz=None):
        arrs = [_d(a) for a in (rho, ux, uy, uz)]
        for a, _ in arrs:
            assert a is None or a.shape == self.shape
        self._chk(self._lib.oracle_set_macros(C.c_void_p(self._h), *[p for _, p in arrs]), "set_macros")

    def set_thermal(self, alpha, gbeta=0.0, theta_ref=0.0):
        self._chk(self._lib.oracle_set_thermal(C.c_void_p(self._h), float(alpha), float(gbeta), float(theta_ref)),
                  "set_thermal")

    def set_inlet_theta(self, theta_b):
        """Prescribed temperature of the EQ_FIXED cells by level, theta_b[nz] (thermal lattice on open faces)."""
        t, tp = _d(np.asarray(theta_b, dtype=np.float64).reshape(self.nz))
        self._chk(self._lib.oracle_set_inlet_theta(C.c_void_p(self._h), tp), "set_inlet_theta")

    def set_thermal_walls(self, on, theta_w):
        """Hold WALL faces (order x-,x+,y-,y+,z-,z+) with on[k] != 0 at temperature theta_w[k] (anti-bounce-back)."""
        a = np.ascontiguousarray(on, dtype=np.int32).reshape(6)
        t, tp = _d(np.asarray(theta_w, dtype=np.float64).reshape(6))
        self._chk(self._lib.oracle_set_thermal_walls(C.c_void_p(self._h), a.ctypes.data_as(C.c_void_p), tp), "set_thermal_walls")

    def set_theta(self, theta=None, ux=None, uy=None, uz=None):
        arrs = [_d(a) for a in (theta, ux, uy, uz)]
        for a, _ in arrs:
            assert a is None or a.shape == self.shape
        self._chk(self._lib.oracle_set_theta(C.c_void_p(self._h), *[p for _, p in arrs]), "set_theta")

    def get_theta(self):
        out = np.zeros(self.shape)
        self._chk(self._lib.oracle_get_theta(C.c_void_p(self._h), out.ctypes.data_as(C.c_void_p)), "get_theta")
        return out

    def get_thermal_state(self):
        """the 7 thermal populations of the stored state, [7][nz][ny][nx]"""
        out = np.zeros((7,) + self.shape)
        self._chk(self._lib.oracle_get_thermal_state(C.c_void_p(self._h), out.ctypes.data_as(C.c_void_p)), "get_thermal_state")
        return out

    def step(self, n=1):
        self._chk(self._lib.oracle_step(C.c_void_p(self._h), int(n)), "step")

    def get_macros(self):
        out = [np.zeros(self.shape) for _ in range(4)]
        self._chk(self._lib.oracle_get_macros(C.c_void_p(self._h), *[a.ctypes.data_as(C.c_void_p) for a in out]),
                  "get_macros")
        return tuple(out)

    def mean_config(self, start_step, every):
        self._chk(self._lib.oracle_mean_config(C.c_void_p(self._h), C.c_long(start_step), int(every)), "mean_config")

    def mean_reset(self):
        self._chk(self._lib.oracle_mean_reset(C.c_void_p(self._h)), "mean_reset")

    def get_mean(self):
        out = [np.zeros(self.shape) for _ in range(3)]
        n = C.c_long()
        self._chk(self._lib.oracle_get_mean(C.c_void_p(self._h), *[a.ctypes.data_as(C.c_void_p) for a in out],
                                            C.byref(n)), "get_mean")
        return out[0], out[1], out[2], n.value

    def get_state(self):
        out = np.zeros((19,) + self.shape)
        self._chk(self._lib.oracle_get_state(C.c_void_p(self._h), out.ctypes.data_as(C.c_void_p)), "get_state")
        return out

    def set_state(self, f):
        f, p = _d(f)
        assert f.shape == (19,) + self.shape
        self._chk(self._lib.oracle_set_state(C.c_void_p(self._h), p), "set_state")

    def get_step(self):
        return int(self._lib.oracle_get_step(C.c_void_p(self._h)))

    def set_step(self, s):
        self._lib.oracle_set_step(C.c_void_p(self._h), C.c_long(s))

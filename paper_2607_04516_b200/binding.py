"""Thin Python binding of the C-ABI library (include/lbm.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of ``liblbm_b200.so``.  PyTorch is used for device memory (the
workspace and output tensors) and for the stream; numpy arrays are passed as HOST pointers (the library copies
them).  There is no CPU fallback: if the library has not been built, or no CUDA device exists, the binding raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liblbm_b200.so")
_lib = None

PERIODIC, WALL, FREE_SLIP, EQ_FIXED, EQ_OUTFLOW = 0, 1, 2, 3, 4
FLUID, SOLID, CELL_EQ_FIXED, CELL_EQ_OUTFLOW = 0, 1, 2, 3
_ERR = {-1: "LBM_EINVAL", -2: "LBM_ENOMEM", -3: "LBM_ECUDA", -4: "LBM_ESTATE"}

# every symbol include/lbm.h declares (tests check that the .so exports them all)
SYMBOLS = [
    "lbm_workspace_bytes", "lbm_create", "lbm_create_ex", "lbm_destroy", "lbm_set_boundaries", "lbm_set_flags",
    "lbm_set_inlet_profile", "lbm_set_inlet_profile_f64", "lbm_set_inlet_plane", "lbm_set_inlet_plane_f64",
    "lbm_feed_inlet", "lbm_set_macros", "lbm_set_macros_f64", "lbm_step", "lbm_mean_config", "lbm_mean_reset",
    "lbm_get_macros", "lbm_get_macros_f64", "lbm_get_mean", "lbm_get_mean_f64", "lbm_get_flags", "lbm_get_links",
    "lbm_get_state", "lbm_set_state", "lbm_get_state_box", "lbm_set_state_box", "lbm_get_macros_box", "lbm_get_macros_box_f64", "lbm_get_mean_box", "lbm_get_step", "lbm_set_step", "lbm_sync", "lbm_last_error",
    "lbm_launch_count", "lbm_lattice", "lbm_set_variant", "lbm_set_coriolis", "lbm_balance_flux",
    "lbm_set_damping", "lbm_set_inflow_turbulence", "lbm_set_flags_mask", "lbm_set_flags_mesh",
    "lbm_set_thermal", "lbm_set_theta", "lbm_set_theta_f64", "lbm_get_theta", "lbm_get_theta_f64",
    "lbm_get_thermal_state", "lbm_set_thermal_state", "lbm_set_thermal_walls", "lbm_set_inlet_theta", "lbm_set_inlet_theta_f64",
    "lbm_voxelise_mesh_static",
]


class LbmError(RuntimeError):
    pass


def library_path() -> str:
    return _SO


def load_library():
    """dlopen the in-tree CUDA library.  Raises if it is missing — there is no fallback path."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_SO):
        raise LbmError(f"{_SO} not built: run `python -m paper_2607_04516_b200.build` (needs nvcc). "
                       "There is no CPU fallback.")
    lib = C.CDLL(_SO)
    vp, i, d, l = C.c_void_p, C.c_int, C.c_double, C.c_long
    lib.lbm_workspace_bytes.argtypes = [i, i, i, i, i, C.POINTER(C.c_size_t)]
    lib.lbm_create.argtypes = [i, i, i, d, d, d, vp, C.POINTER(vp)]
    lib.lbm_create_ex.argtypes = [i, i, i, d, d, d, vp, vp, C.c_size_t, vp, i, i, C.POINTER(vp)]
    lib.lbm_destroy.argtypes = [vp]
    lib.lbm_set_boundaries.argtypes = [vp, vp]
    lib.lbm_set_coriolis.argtypes = [vp, vp]
    lib.lbm_balance_flux.argtypes = [vp, vp, vp]
    lib.lbm_set_damping.argtypes = [vp, vp, vp, vp]
    lib.lbm_set_inflow_turbulence.argtypes = [vp, i, vp, C.c_double, C.c_double, C.c_double]
    lib.lbm_set_flags.argtypes = [vp, vp]
    lib.lbm_set_flags_mask.argtypes = [vp, vp, vp]
    lib.lbm_set_flags_mesh.argtypes = [vp, vp, i, vp, i]
    for n in ("lbm_set_inlet_profile", "lbm_set_inlet_profile_f64"):
        getattr(lib, n).argtypes = [vp, vp, vp, vp]
    for n in ("lbm_set_inlet_plane", "lbm_set_inlet_plane_f64"):
        getattr(lib, n).argtypes = [vp, i, vp]
    lib.lbm_feed_inlet.argtypes = [vp, vp, i]
    for n in ("lbm_set_macros", "lbm_set_macros_f64", "lbm_get_macros", "lbm_get_macros_f64"):
        getattr(lib, n).argtypes = [vp, vp, vp, vp, vp]
    lib.lbm_step.argtypes = [vp, i]
    lib.lbm_set_thermal.argtypes = [vp, C.c_double, C.c_double, C.c_double]
    for n in ("lbm_set_theta", "lbm_set_theta_f64"):
        getattr(lib, n).argtypes = [vp, vp, vp, vp, vp]
    for n in ("lbm_get_theta", "lbm_get_theta_f64", "lbm_get_thermal_state", "lbm_set_thermal_state", "lbm_set_inlet_theta",
              "lbm_set_inlet_theta_f64"):
        getattr(lib, n).argtypes = [vp, vp]
    lib.lbm_set_thermal_walls.argtypes = [vp, vp, vp]
    lib.lbm_mean_config.argtypes = [vp, l, i]
    lib.lbm_mean_reset.argtypes = [vp]
    for n in ("lbm_get_mean", "lbm_get_mean_f64"):
        getattr(lib, n).argtypes = [vp, vp, vp, vp, C.POINTER(l)]
    lib.lbm_get_flags.argtypes = [vp, vp]
    lib.lbm_get_links.argtypes = [vp, vp]
    lib.lbm_get_state.argtypes = [vp, vp]
    lib.lbm_set_state.argtypes = [vp, vp]
    lib.lbm_get_state_box.argtypes = [vp, vp, vp, vp]
    lib.lbm_set_state_box.argtypes = [vp, vp, vp, vp]
    lib.lbm_get_macros_box.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.lbm_get_macros_box_f64.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.lbm_get_mean_box.argtypes = [vp, vp, vp, vp, vp, vp, C.POINTER(C.c_long)]
    lib.lbm_get_step.argtypes = [vp]
    lib.lbm_get_step.restype = l
    lib.lbm_set_step.argtypes = [vp, l]
    lib.lbm_sync.argtypes = [vp]
    lib.lbm_last_error.argtypes = [vp]
    lib.lbm_last_error.restype = C.c_char_p
    lib.lbm_launch_count.argtypes = [vp]
    lib.lbm_launch_count.restype = l
    lib.lbm_lattice.argtypes = [vp, vp]
    lib.lbm_set_variant.argtypes = [vp, i]
    lib.lbm_voxelise_mesh_static.argtypes = [i, i, i, i, vp, i, vp, vp, C.c_char_p, C.c_size_t]
    _lib = lib
    return lib


def _ptr(a, dtype):
    """Pointer of a numpy array (host) or torch tensor (host or device); None -> NULL.  Returns (keepalive, ptr)."""
    if a is None:
        return None, None
    if isinstance(a, np.ndarray):
        a = np.ascontiguousarray(a, dtype=dtype)
        return a, a.ctypes.data
    import torch
    if isinstance(a, torch.Tensor):
        want = {np.float32: torch.float32, np.float64: torch.float64, np.int32: torch.int32,
                np.uint8: torch.uint8, np.uint32: torch.int32}[dtype]
        if a.dtype != want or not a.is_contiguous():
            a = a.to(want).contiguous()
        return a, a.data_ptr()
    a = np.ascontiguousarray(a, dtype=dtype)
    return a, a.ctypes.data


PREC_F32, PREC_F64, PREC_F32_S16 = 0, 1, 2   # include/lbm.h LBM_PREC_*
STREAM_INPLACE = 16                           # include/lbm.h LBM_STREAM_INPLACE (OR-ed into the precision argument)
STATIC_VOXEL_MAX_CELLS = 2097152              # include/lbm.h LBM_STATIC_VOXEL_MAX_CELLS


def voxelise_mesh_static(tri, nx, ny, nz, min_votes=2, out=None, stream=None):
    """lbm_voxelise_mesh_static: the mesh voxeliser without a handle and without any allocation inside the library (its
    scratch is a static device array; boxes of at most STATIC_VOXEL_MAX_CELLS cells; overlapping calls race).
    tri: DEVICE float32 tensor [n][3][3]; out: DEVICE uint8 tensor [nz][ny][nx] (allocated here, by torch, if None).
    Runs on the device of `tri`.  Returns out (1 = SOLID)."""
    import torch
    lib = load_library()
    if not (isinstance(tri, torch.Tensor) and tri.is_cuda and tri.dtype == torch.float32 and tri.is_contiguous()):
        raise ValueError("tri must be a contiguous float32 CUDA tensor [n][3][3] (host arrays are refused: no staging, no allocation)")
    n_tri = int(tri.numel() // 9)
    with torch.cuda.device(tri.device):
        if out is None:
            out = torch.empty((int(nz), int(ny), int(nx)), dtype=torch.uint8, device=tri.device)
        st = stream if stream is not None else torch.cuda.current_stream(tri.device)
        err = C.create_string_buffer(256)
        rc = lib.lbm_voxelise_mesh_static(int(nx), int(ny), int(nz), n_tri, tri.data_ptr() if n_tri else None, int(min_votes),
                                          out.data_ptr(), st.cuda_stream, err, 256)
    if rc != 0:
        raise LbmError(f"lbm_voxelise_mesh_static failed: {_ERR.get(rc, rc)}: {err.value.decode()}")
    return out


class Lbm:
    """One lattice on one GPU.  Same call names as include/lbm.h without the ``lbm_`` prefix."""

    def __init__(self, nx, ny, nz, nu0, Cs=0.0, f_cor=0.0, F=(0.0, 0.0, 0.0), faces=None, fp64=False,
                 want_mean=True, device="cuda:0", stream=None, storage16=False, inplace=False, guard_bytes=0):
        import torch
        if not torch.cuda.is_available():
            raise LbmError("no CUDA device: the LBM path has no CPU fallback")
        self._lib = load_library()
        self._torch = torch
        self.device = torch.device(device)
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.shape = (self.nz, self.ny, self.nx)
        self.fp64 = bool(fp64)
        self.storage16 = bool(storage16)
        if fp64 and storage16:
            raise ValueError("fp64 and storage16 exclude each other")
        precision = PREC_F64 if fp64 else (PREC_F32_S16 if storage16 else PREC_F32)     # include/lbm.h LBM_PREC_*
        self.inplace = bool(inplace)
        if inplace:
            precision |= STREAM_INPLACE                                                  # include/lbm.h LBM_STREAM_INPLACE
        F = np.atleast_1d(np.asarray(F, dtype=np.float64))
        if F.size == 1:
            F = np.array([F[0], 0.0, 0.0])
        nbytes = C.c_size_t()
        self._chk0(self._lib.lbm_workspace_bytes(self.nx, self.ny, self.nz, int(want_mean), precision, C.byref(nbytes)),
                   "workspace_bytes")
        with torch.cuda.device(self.device):
            # guard_bytes > 0 (tests): the workspace handed to the library sits between two bands filled with 0xA5, which
            # guards_intact() inspects — a store of any kernel outside its workspace shows up there
            self._guard = int(guard_bytes) // 256 * 256
            self._ws = torch.full((nbytes.value + 512 + 2 * self._guard,), 0xA5, dtype=torch.uint8, device=self.device)
            base = self._ws.data_ptr()
            aligned = (base + 255) // 256 * 256 + self._guard
            self._ws_off = aligned - base
            self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = C.c_void_p()
            rc = self._lib.lbm_create_ex(self.nx, self.ny, self.nz, float(nu0), float(Cs), float(f_cor), F.ctypes.data,
                                         aligned, nbytes.value, self._stream.cuda_stream, precision, int(want_mean),
                                         C.byref(h))
        self._chk0(rc, "create_ex")
        self._h = h
        self.workspace_bytes = nbytes.value
        if faces is not None:
            self.set_boundaries(faces)

    # -- plumbing
    def _chk0(self, rc, what):
        if rc != 0:
            raise LbmError(f"lbm_{what} failed: {_ERR.get(rc, rc)}")

    def _chk(self, rc, what):
        if rc != 0:
            msg = self._lib.lbm_last_error(self._h)
            raise LbmError(f"lbm_{what} failed: {_ERR.get(rc, rc)}: {msg.decode() if msg else ''}")

    def guards_intact(self) -> bool:
        """True if no byte outside the workspace handed to the library (guard bands before and after it) has been written."""
        lo = self._ws[: self._ws_off]
        hi = self._ws[self._ws_off + self.workspace_bytes:]
        return bool((lo == 0xA5).all().item()) and bool((hi == 0xA5).all().item())

    def close(self):
        if getattr(self, "_h", None):
            self._lib.lbm_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _new(self, dtype, shape=None):
        t = self._torch
        return t.empty(shape or self.shape, dtype=dtype, device=self.device)

    # -- setup
    def set_boundaries(self, faces):
        a = np.ascontiguousarray(faces, dtype=np.int32)
        if a.shape != (6,):
            raise ValueError("faces must have 6 entries")
        self._chk(self._lib.lbm_set_boundaries(self._h, a.ctypes.data), "set_boundaries")

    def set_coriolis(self, f):
        """Full Coriolis vector f = 2 Omega in lattice units; (0, 0, f_cor) is the scalar form of the constructor."""
        a = np.ascontiguousarray(f, dtype=np.float64)
        if a.shape != (3,):
            raise ValueError("f must have 3 entries")
        self._chk(self._lib.lbm_set_coriolis(self._h, a.ctypes.data), "set_coriolis")

    def set_damping(self, width, peak, target=None):
        """Sponge / buffer zones: per-face width (cells) and peak coefficient, host target profile [3][nz]."""
        w = np.ascontiguousarray(width, dtype=np.int32)
        pk = np.ascontiguousarray(peak, dtype=np.float64)
        if w.shape != (6,) or pk.shape != (6,):
            raise ValueError("width and peak must have 6 entries")
        t = None
        if target is not None:
            t = np.ascontiguousarray(target, dtype=np.float64)
            if t.shape != (3, self.nz):
                raise ValueError("target must be [3][nz]")
        self._chk(self._lib.lbm_set_damping(self._h, w.ctypes.data, pk.ctypes.data, t.ctypes.data if t is not None else None),
                  "set_damping")

    def set_inflow_turbulence(self, modes, u_rms=0.0, k_e=1.0, k_eta=0.0):
        """Synthetic von Karman fluctuations on active inflow cells; host table [n][9] = kappa, sigma, psi, omega,
        dkappa (None / empty: off)."""
        if modes is None or len(modes) == 0:
            self._chk(self._lib.lbm_set_inflow_turbulence(self._h, 0, None, 0.0, 1.0, 0.0), "set_inflow_turbulence")
            return
        m = np.ascontiguousarray(modes, dtype=np.float64)
        if m.ndim != 2 or m.shape[1] != 9:
            raise ValueError("modes must be [n][9]")
        self._chk(self._lib.lbm_set_inflow_turbulence(self._h, m.shape[0], m.ctypes.data, float(u_rms), float(k_e), float(k_eta)),
                  "set_inflow_turbulence")

    def balance_flux(self):
        """Global flux-balancing correction of the EQ_FIXED face velocities; returns (flux_before, flux_after)."""
        a, b = C.c_double(), C.c_double()
        self._chk(self._lib.lbm_balance_flux(self._h, C.addressof(a), C.addressof(b)), "balance_flux")
        return a.value, b.value

    def set_flags(self, height=None):
        k, p = _ptr(height, np.int32)
        if k is not None and tuple(k.shape) != (self.ny, self.nx):
            raise ValueError("height must be [ny][nx]")
        self._chk(self._lib.lbm_set_flags(self._h, p), "set_flags")

    def set_flags_mask(self, height=None, solid=None):
        """Heightmap (or None) merged with a general solid mask uint8 [nz][ny][nx] (host or device)."""
        k, p = _ptr(height, np.int32)
        if k is not None and tuple(k.shape) != (self.ny, self.nx):
            raise ValueError("height must be [ny][nx]")
        m, mp = _ptr(solid, np.uint8)
        if m is not None and tuple(m.shape) != self.shape:
            raise ValueError("solid must be [nz][ny][nx]")
        self._chk(self._lib.lbm_set_flags_mask(self._h, p, mp), "set_flags_mask")

    def set_flags_mesh(self, tri, height=None, min_votes=2):
        """Voxelise a triangle mesh float32 [n][3][3] (lattice units, host or device) and merge it with the heightmap."""
        k, p = _ptr(height, np.int32)
        if k is not None and tuple(k.shape) != (self.ny, self.nx):
            raise ValueError("height must be [ny][nx]")
        t, tp = _ptr(tri, np.float32)
        n = 0 if t is None else int(np.prod(tuple(t.shape))) // 9
        if t is not None and int(np.prod(tuple(t.shape))) != 9 * n:
            raise ValueError("tri must be [n][3][3]")
        self._chk(self._lib.lbm_set_flags_mesh(self._h, p, n, tp, int(min_votes)), "set_flags_mesh")

    def set_inlet_profile(self, u, v=None, w=None, f64=False):
        dt = np.float64 if f64 else np.float32
        ks = [_ptr(a, dt) for a in (u, v, w)]
        fn = self._lib.lbm_set_inlet_profile_f64 if f64 else self._lib.lbm_set_inlet_profile
        self._chk(fn(self._h, *[p for _, p in ks]), "set_inlet_profile")

    def set_inlet_plane(self, face, uvw, f64=False):
        k, p = _ptr(uvw, np.float64 if f64 else np.float32)
        fn = self._lib.lbm_set_inlet_plane_f64 if f64 else self._lib.lbm_set_inlet_plane
        self._chk(fn(self._h, int(face), p), "set_inlet_plane")

    def feed_inlet(self, src: "Lbm", src_x_plane: int):
        self._chk(self._lib.lbm_feed_inlet(self._h, src._h, int(src_x_plane)), "feed_inlet")

    def set_macros(self, rho=None, ux=None, uy=None, uz=None, f64=False):
        dt = np.float64 if f64 else np.float32
        ks = [_ptr(a, dt) for a in (rho, ux, uy, uz)]
        for k, _ in ks:
            if k is not None and tuple(k.shape) != self.shape:
                raise ValueError("fields must be [nz][ny][nx]")
        fn = self._lib.lbm_set_macros_f64 if f64 else self._lib.lbm_set_macros
        self._chk(fn(self._h, *[p for _, p in ks]), "set_macros")

    # -- thermal lattice + Boussinesq coupling
    def set_thermal(self, alpha, g_beta=0.0, theta_ref=0.0):
        self._chk(self._lib.lbm_set_thermal(self._h, float(alpha), float(g_beta), float(theta_ref)), "set_thermal")

    def set_theta(self, theta=None, ux=None, uy=None, uz=None, f64=False):
        dt = np.float64 if f64 else np.float32
        ks = [_ptr(a, dt) for a in (theta, ux, uy, uz)]
        for k, _ in ks:
            if k is not None and tuple(k.shape) != self.shape:
                raise ValueError("fields must be [nz][ny][nx]")
        fn = self._lib.lbm_set_theta_f64 if f64 else self._lib.lbm_set_theta
        self._chk(fn(self._h, *[p for _, p in ks]), "set_theta")

    def get_theta(self, out=None, f64=False):
        t = self._torch
        fn = self._lib.lbm_get_theta_f64 if f64 else self._lib.lbm_get_theta
        if out == "host":
            a = np.empty(self.shape, dtype=np.float64 if f64 else np.float32)
            self._chk(fn(self._h, a.ctypes.data), "get_theta")
            return a
        a = out if out is not None else self._new(t.float64 if f64 else t.float32)
        self._chk(fn(self._h, a.data_ptr()), "get_theta")
        return a

    def set_inlet_theta(self, theta_b, f64=False):
        """Prescribed temperature of the EQ_FIXED cells by level, theta_b[nz] (thermal lattice on open faces)."""
        k, p = _ptr(theta_b, np.float64 if f64 else np.float32)
        if tuple(k.shape) != (self.nz,):
            raise ValueError("theta_b must have nz entries")
        fn = self._lib.lbm_set_inlet_theta_f64 if f64 else self._lib.lbm_set_inlet_theta
        self._chk(fn(self._h, p), "set_inlet_theta")

    def set_thermal_walls(self, on, theta_w):
        """Hold WALL faces (order x-,x+,y-,y+,z-,z+) with on[k] != 0 at temperature theta_w[k]."""
        a = np.ascontiguousarray(on, dtype=np.int32)
        t = np.ascontiguousarray(theta_w, dtype=np.float64)
        if a.shape != (6,) or t.shape != (6,):
            raise ValueError("on and theta_w must have 6 entries")
        self._chk(self._lib.lbm_set_thermal_walls(self._h, a.ctypes.data, t.ctypes.data), "set_thermal_walls")

    def get_thermal_state(self):
        """The 7 thermal populations [7][nz][ny][nx] float64 (host): the thermal half of a checkpoint."""
        a = np.empty((7,) + self.shape, dtype=np.float64)
        self._chk(self._lib.lbm_get_thermal_state(self._h, a.ctypes.data), "get_thermal_state")
        return a

    def set_thermal_state(self, hpop):
        k, p = _ptr(hpop, np.float64)
        if tuple(k.shape) != (7,) + self.shape:
            raise ValueError("thermal state must be [7][nz][ny][nx]")
        self._chk(self._lib.lbm_set_thermal_state(self._h, p), "set_thermal_state")

    # -- the hot call
    def step(self, n=1):
        self._chk(self._lib.lbm_step(self._h, int(n)), "step")

    def mean_config(self, start_step, every):
        self._chk(self._lib.lbm_mean_config(self._h, int(start_step), int(every)), "mean_config")

    def mean_reset(self):
        self._chk(self._lib.lbm_mean_reset(self._h), "mean_reset")

    # -- results.  out=None: fresh torch device tensors; out="host": numpy arrays filled through HOST pointers
    def get_macros(self, out=None, f64=False):
        t = self._torch
        fn = self._lib.lbm_get_macros_f64 if f64 else self._lib.lbm_get_macros
        if out == "host":
            arrs = [np.empty(self.shape, dtype=np.float64 if f64 else np.float32) for _ in range(4)]
            self._chk(fn(self._h, *[a.ctypes.data for a in arrs]), "get_macros")
            return tuple(arrs)
        arrs = out if out is not None else [self._new(t.float64 if f64 else t.float32) for _ in range(4)]
        self._chk(fn(self._h, *[a.data_ptr() if a is not None else None for a in arrs]), "get_macros")
        return tuple(arrs)

    def get_mean(self, out=None, f64=False):
        t = self._torch
        fn = self._lib.lbm_get_mean_f64 if f64 else self._lib.lbm_get_mean
        n = C.c_long()
        if out == "host":
            arrs = [np.empty(self.shape, dtype=np.float64 if f64 else np.float32) for _ in range(3)]
            self._chk(fn(self._h, *[a.ctypes.data for a in arrs], C.byref(n)), "get_mean")
            return arrs[0], arrs[1], arrs[2], n.value
        arrs = out if out is not None else [self._new(t.float64 if f64 else t.float32) for _ in range(3)]
        self._chk(fn(self._h, *[a.data_ptr() for a in arrs], C.byref(n)), "get_mean")
        return arrs[0], arrs[1], arrs[2], n.value

    def get_flags(self):
        out = np.empty(self.shape, dtype=np.uint8)
        self._chk(self._lib.lbm_get_flags(self._h, out.ctypes.data), "get_flags")
        return out

    def get_links(self):
        out = np.empty(self.shape, dtype=np.uint32)
        self._chk(self._lib.lbm_get_links(self._h, out.ctypes.data), "get_links")
        return out

    def get_state(self, out=None):
        if out == "host":
            a = np.empty((19,) + self.shape, dtype=np.float64)
            self._chk(self._lib.lbm_get_state(self._h, a.ctypes.data), "get_state")
            return a
        a = self._new(self._torch.float64, (19,) + self.shape)
        self._chk(self._lib.lbm_get_state(self._h, a.data_ptr()), "get_state")
        return a

    def set_state(self, f):
        k, p = _ptr(f, np.float64)
        if tuple(k.shape) != (19,) + self.shape:
            raise ValueError("state must be [19][nz][ny][nx]")
        self._chk(self._lib.lbm_set_state(self._h, p), "set_state")

    def _box(self, lo, hi):
        lo = np.ascontiguousarray(lo, dtype=np.int32)
        hi = np.ascontiguousarray(hi, dtype=np.int32)
        if lo.shape != (3,) or hi.shape != (3,):
            raise ValueError("lo and hi must be (x, y, z)")
        return lo, hi

    def get_state_box(self, lo, hi, out=None):
        """populations of the box lo <= (x, y, z) < hi: [19][hi_z-lo_z][hi_y-lo_y][hi_x-lo_x] float64"""
        lo, hi = self._box(lo, hi)
        shape = (19, max(int(hi[2] - lo[2]), 0), max(int(hi[1] - lo[1]), 0), max(int(hi[0] - lo[0]), 0))
        if out == "host":
            a = np.empty(shape, dtype=np.float64)
            self._chk(self._lib.lbm_get_state_box(self._h, lo.ctypes.data, hi.ctypes.data, a.ctypes.data), "get_state_box")
            return a
        a = self._new(self._torch.float64, shape)
        self._chk(self._lib.lbm_get_state_box(self._h, lo.ctypes.data, hi.ctypes.data, a.data_ptr()), "get_state_box")
        return a

    def get_macros_box(self, lo, hi, f64=False):
        """rho, ux, uy, uz of the box lo <= (x, y, z) < hi: device tensors [hi_z-lo_z][hi_y-lo_y][hi_x-lo_x]"""
        lo, hi = self._box(lo, hi)
        t = self._torch
        shape = (max(int(hi[2] - lo[2]), 1), max(int(hi[1] - lo[1]), 1), max(int(hi[0] - lo[0]), 1))
        arrs = [self._new(t.float64 if f64 else t.float32, shape) for _ in range(4)]
        fn = self._lib.lbm_get_macros_box_f64 if f64 else self._lib.lbm_get_macros_box
        self._chk(fn(self._h, lo.ctypes.data, hi.ctypes.data, *[a.data_ptr() for a in arrs]), "get_macros_box")
        return tuple(arrs)

    def get_mean_box(self, lo, hi):
        lo, hi = self._box(lo, hi)
        shape = (max(int(hi[2] - lo[2]), 1), max(int(hi[1] - lo[1]), 1), max(int(hi[0] - lo[0]), 1))
        arrs = [self._new(self._torch.float32, shape) for _ in range(3)]
        n = C.c_long()
        self._chk(self._lib.lbm_get_mean_box(self._h, lo.ctypes.data, hi.ctypes.data, *[a.data_ptr() for a in arrs], C.byref(n)), "get_mean_box")
        return arrs[0], arrs[1], arrs[2], n.value

    def set_state_box(self, lo, hi, f):
        lo, hi = self._box(lo, hi)
        k, p = _ptr(f, np.float64)
        if tuple(k.shape) != (19, int(hi[2] - lo[2]), int(hi[1] - lo[1]), int(hi[0] - lo[0])):
            raise ValueError("state must be [19][hi_z-lo_z][hi_y-lo_y][hi_x-lo_x]")
        self._chk(self._lib.lbm_set_state_box(self._h, lo.ctypes.data, hi.ctypes.data, p), "set_state_box")

    def get_step(self):
        return int(self._lib.lbm_get_step(self._h))

    def set_step(self, s):
        self._chk(self._lib.lbm_set_step(self._h, int(s)), "set_step")

    def sync(self):
        self._chk(self._lib.lbm_sync(self._h), "sync")

    def launch_count(self):
        return int(self._lib.lbm_launch_count(self._h))

    def set_variant(self, v):
        self._chk(self._lib.lbm_set_variant(self._h, int(v)), "set_variant")

    @property
    def cuda_stream(self):
        return self._stream


def lattice():
    lib = load_library()
    c = np.zeros((19, 3), dtype=np.int32)
    opp = np.zeros(19, dtype=np.int32)
    rc = lib.lbm_lattice(c.ctypes.data, opp.ctypes.data)
    if rc != 0:
        raise LbmError("lbm_lattice failed")
    return c, opp


def from_workload(wl, fp64=False, want_mean=True, device="cuda:0", storage16=False, stream=None, inplace=False) -> Lbm:
    """Create a handle for a workloads.Workload and load its flags, inlet profile and initial field."""
    sim = Lbm(wl.nx, wl.ny, wl.nz, wl.nu0, wl.Cs, wl.f_cor, wl.F, wl.faces, fp64=fp64, want_mean=want_mean,
              device=device, storage16=storage16, stream=stream, inplace=inplace)
    sim.set_flags(wl.height)
    if wl.inlet_profile is not None:
        sim.set_inlet_profile(*wl.inlet_profile)
    if wl.init is not None:
        sim.set_macros(*wl.init)
    else:
        sim.set_macros()
    if wl.extra.get("thermal") is not None:
        sim.set_thermal(*wl.extra["thermal"])
        sim.set_theta(wl.extra.get("theta"))
    return sim

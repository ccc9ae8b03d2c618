"""Thin Python binding of the C ABI in include/clvisc_hydro.h (argument marshalling only).

PyTorch supplies device memory (the workspace and the field tensors) and the CUDA stream; every step
of the path runs in the kernels of libclvisc_hydro.so.  There is no CPU fallback: if the library is
missing and cannot be built, or no CUDA device is usable, the calls raise.
"""
from __future__ import annotations

import ctypes
from ctypes import POINTER, Structure, byref, c_double, c_int, c_longlong, c_size_t, c_void_p

import numpy as np

from . import build as _build

HYDRO_MEM_DEVICE, HYDRO_MEM_HOST = 0, 1
SYMBOLS = ["hydro_workspace_bytes", "hydro_create", "hydro_load", "hydro_set_history", "hydro_read_history",
           "hydro_step", "hydro_read", "hydro_diag", "hydro_launch_count", "hydro_kernel", "hydro_destroy", "hydro_strerror",
           "hydro_freezeout_bytes", "hydro_freezeout_begin", "hydro_freezeout_slab", "hydro_freezeout_run",
           "hydro_workspace_bytes_ext", "hydro_load_ext", "hydro_read_ext", "hydro_eos_e_of_temperature",
           "hydro_stage", "hydro_plane_bytes", "hydro_planes"]


class hydro_grid(Structure):
    _fields_ = [("nx", c_int), ("ny", c_int), ("nz", c_int), ("dx", c_double), ("dy", c_double),
                ("deta", c_double), ("bc", c_int * 3), ("geometry", c_int)]


class hydro_eos(Structure):
    _fields_ = [("kind", c_int), ("n", c_int), ("e_min", c_double), ("e_max", c_double),
                ("P", POINTER(c_double)), ("T", POINTER(c_double)), ("c_sb", c_double)]


class hydro_opts(Structure):
    _fields_ = [("precision", c_int), ("minmod_theta", c_double), ("e_floor", c_double),
                ("pi_limit_xi", c_double), ("v_max", c_double), ("root_iters", c_int), ("kernel", c_int),
                ("stream", c_void_p), ("workspace", c_void_p), ("workspace_bytes", c_size_t),
                ("lambda1_hat", c_double), ("tau_pi_coeff", c_double), ("strict_eq53", c_int),
                ("bulk_baryon", c_int), ("zeta_over_s", c_double)]


class hydro_diag_t(Structure):
    _fields_ = [("tau", c_double), ("step", c_longlong), ("cfl", c_double * 3), ("e_max", c_double),
                ("n_floor", c_longlong), ("n_clamp", c_longlong), ("n_pi_limited", c_longlong),
                ("n_nan", c_longlong), ("n_root_unconverged", c_longlong)]


_lib = None


def load_library():
    """dlopen libclvisc_hydro.so (building it first when stale and nvcc is present)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    lib = ctypes.CDLL(path)
    lib.hydro_workspace_bytes.restype = c_size_t
    lib.hydro_workspace_bytes.argtypes = [POINTER(hydro_grid), c_int, c_double]
    lib.hydro_create.restype = c_int
    lib.hydro_create.argtypes = [POINTER(c_void_p), POINTER(hydro_grid), c_double, c_double,
                                 POINTER(hydro_eos), c_double, POINTER(hydro_opts)]
    lib.hydro_load.restype = c_int
    lib.hydro_load.argtypes = [c_void_p, c_void_p, c_void_p, c_int]
    lib.hydro_set_history.restype = c_int
    lib.hydro_set_history.argtypes = [c_void_p, c_void_p, c_int]
    lib.hydro_read_history.restype = c_int
    lib.hydro_read_history.argtypes = [c_void_p, c_void_p, c_int]
    lib.hydro_step.restype = c_int
    lib.hydro_step.argtypes = [c_void_p, c_int]
    lib.hydro_read.restype = c_int
    lib.hydro_read.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_int]
    lib.hydro_diag.restype = c_int
    lib.hydro_diag.argtypes = [c_void_p, POINTER(hydro_diag_t)]
    lib.hydro_launch_count.restype = c_longlong
    lib.hydro_launch_count.argtypes = [c_void_p]
    lib.hydro_kernel.restype = c_int
    lib.hydro_kernel.argtypes = [c_void_p]
    lib.hydro_freezeout_bytes.restype = c_size_t
    lib.hydro_freezeout_bytes.argtypes = [POINTER(hydro_grid), c_int]
    lib.hydro_freezeout_begin.restype = c_int
    lib.hydro_freezeout_begin.argtypes = [c_void_p, c_void_p, c_size_t, c_double]
    lib.hydro_freezeout_slab.restype = c_int
    lib.hydro_freezeout_slab.argtypes = [c_void_p, c_void_p, c_void_p, c_longlong, POINTER(c_longlong),
                                         POINTER(c_longlong)]
    lib.hydro_freezeout_run.restype = c_int
    lib.hydro_freezeout_run.argtypes = [c_void_p, c_int, c_int, c_void_p, c_void_p, c_longlong, POINTER(c_longlong),
                                        POINTER(c_int)]
    lib.hydro_workspace_bytes_ext.restype = c_size_t
    lib.hydro_workspace_bytes_ext.argtypes = [POINTER(hydro_grid), c_int, c_double, c_int]
    lib.hydro_load_ext.restype = c_int
    lib.hydro_load_ext.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_int]
    lib.hydro_read_ext.restype = c_int
    lib.hydro_read_ext.argtypes = [c_void_p, c_void_p, c_void_p, c_int]
    lib.hydro_eos_e_of_temperature.restype = c_int
    lib.hydro_eos_e_of_temperature.argtypes = [POINTER(hydro_eos), c_double, POINTER(c_double)]
    lib.hydro_stage.restype = c_int
    lib.hydro_stage.argtypes = [c_void_p, c_int]
    lib.hydro_plane_bytes.restype = c_size_t
    lib.hydro_plane_bytes.argtypes = [c_void_p]
    lib.hydro_planes.restype = c_int
    lib.hydro_planes.argtypes = [c_void_p, c_int, c_int, c_int, c_void_p, c_int, c_int]
    lib.hydro_destroy.restype = None
    lib.hydro_destroy.argtypes = [c_void_p]
    lib.hydro_strerror.restype = ctypes.c_char_p
    lib.hydro_strerror.argtypes = [c_int]
    _lib = lib
    return lib


class HydroError(RuntimeError):
    pass


def _check(rc, what):
    if rc < 0:
        raise HydroError(f"{what}: {load_library().hydro_strerror(rc).decode()} (rc={rc})")
    return rc


def make_eos(eos):
    """hydro_eos from an inputs.conformal_eos() / crossover_table() dict; returns (struct, keep-alive arrays)."""
    e = hydro_eos()
    e.kind, e.n, e.e_min, e.e_max, e.c_sb = int(eos["kind"]), int(eos["n"]), float(eos["e_min"]), \
        float(eos["e_max"]), float(eos["c_sb"])
    P = None if eos["P"] is None else np.ascontiguousarray(eos["P"], dtype=np.float64)
    T = None if eos["T"] is None else np.ascontiguousarray(eos["T"], dtype=np.float64)
    e.P = None if P is None else P.ctypes.data_as(POINTER(c_double))
    e.T = None if T is None else T.ctypes.data_as(POINTER(c_double))
    return e, (P, T)


def eos_e_of_T(eos, T_frz: float) -> float:
    """hydro_eos_e_of_temperature: the energy density with temperature T_frz (GeV) -- a constant-T_f freeze-out surface is the
    constant-e surface at this value.  Host arithmetic of the library; needs no device."""
    e, keep = make_eos(eos)
    out = c_double(0.0)
    _check(load_library().hydro_eos_e_of_temperature(byref(e), float(T_frz), byref(out)), "hydro_eos_e_of_temperature")
    return out.value


def make_grid(nx, ny, nz, dx, dy, deta, bc=(0, 0, 0), geometry=0):
    g = hydro_grid()
    g.nx, g.ny, g.nz, g.dx, g.dy, g.deta, g.geometry = nx, ny, nz, dx, dy, deta, geometry
    g.bc[0], g.bc[1], g.bc[2] = bc
    return g


def workspace_bytes(grid: hydro_grid, precision: int, eta_over_s: float) -> int:
    return int(load_library().hydro_workspace_bytes(byref(grid), precision, eta_over_s))


class Hydro:
    """hydro_create / hydro_load / hydro_step / hydro_read / hydro_diag / hydro_destroy.

    eos: dict(kind, n, e_min, e_max, P, T, c_sb) as produced by inputs.conformal_eos() /
    inputs.crossover_table().  Fields are torch CUDA tensors (used in place) or host arrays
    (numpy / CPU tensors, copied inside the call), dtype float64 or float32 to match `precision`.
    """

    def __init__(self, nx, ny, nz, dx, dy, deta, dtau, tau0, eos, eta_over_s, bc=(0, 0, 0), geometry=0,
                 precision=64, minmod_theta=1.1, e_floor=1e-7, pi_limit_xi=1.0, v_max=0.0, root_iters=0,
                 kernel=0, device="cuda:0", stream=None, lambda1_hat=0.0, tau_pi_coeff=0.0, strict_eq53=0,
                 bulk_baryon=0, zeta_over_s=0.0):
        import torch
        self._torch = torch
        self._lib = load_library()
        self._h = c_void_p()
        if not torch.cuda.is_available():
            raise HydroError("no CUDA device: the CLVisc step has no CPU fallback")
        self.device = torch.device(device)
        self.precision = precision
        self.dtype = torch.float64 if precision == 64 else torch.float32
        self.np_dtype = np.float64 if precision == 64 else np.float32
        self.shape = (nz, ny, nx)
        self.N = nx * ny * nz
        self.viscous = eta_over_s > 0
        self.grid = make_grid(nx, ny, nz, dx, dy, deta, bc, geometry)
        self.bulk_baryon = int(bulk_baryon)
        nbytes = int(self._lib.hydro_workspace_bytes_ext(byref(self.grid), precision, eta_over_s, self.bulk_baryon))
        if nbytes == 0:
            raise HydroError("hydro_workspace_bytes: invalid grid / precision")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        base = self.workspace.data_ptr()
        aligned = (base + 255) // 256 * 256
        e = hydro_eos()
        e.kind, e.n, e.e_min, e.e_max, e.c_sb = int(eos["kind"]), int(eos["n"]), float(eos["e_min"]), \
            float(eos["e_max"]), float(eos["c_sb"])
        self._P = None if eos["P"] is None else np.ascontiguousarray(eos["P"], dtype=np.float64)
        self._T = None if eos["T"] is None else np.ascontiguousarray(eos["T"], dtype=np.float64)
        e.P = None if self._P is None else self._P.ctypes.data_as(POINTER(c_double))
        e.T = None if self._T is None else self._T.ctypes.data_as(POINTER(c_double))
        o = hydro_opts()
        o.precision, o.minmod_theta, o.e_floor, o.pi_limit_xi, o.v_max = precision, minmod_theta, e_floor, \
            pi_limit_xi, v_max
        o.root_iters, o.kernel = root_iters, kernel
        o.lambda1_hat, o.tau_pi_coeff = lambda1_hat, tau_pi_coeff
        o.strict_eq53 = int(strict_eq53)
        o.bulk_baryon, o.zeta_over_s = self.bulk_baryon, float(zeta_over_s)
        o.stream = c_void_p(self.stream.cuda_stream)
        o.workspace, o.workspace_bytes = c_void_p(aligned), nbytes
        with torch.cuda.device(self.device):
            _check(self._lib.hydro_create(byref(self._h), byref(self.grid), dtau, tau0, byref(e), eta_over_s,
                                          byref(o)), "hydro_create")

    # -- marshalling helpers ------------------------------------------------------------------
    def _ptr(self, a, ncomp, writable=False):
        """(pointer, mem tag, keep-alive) of a tensor/array with ncomp*N elements of the context dtype."""
        torch = self._torch
        if a is None:
            return None, HYDRO_MEM_DEVICE, None
        if isinstance(a, torch.Tensor):
            if a.dtype != self.dtype or not a.is_contiguous() or a.numel() != ncomp * self.N:
                raise HydroError("tensor must be contiguous, of the context dtype, with %d elements" % (ncomp * self.N))
            return c_void_p(a.data_ptr()), (HYDRO_MEM_DEVICE if a.is_cuda else HYDRO_MEM_HOST), a
        a = np.ascontiguousarray(a, dtype=self.np_dtype) if not writable else a
        if a.dtype != self.np_dtype or not a.flags["C_CONTIGUOUS"] or a.size != ncomp * self.N:
            raise HydroError("array must be C-contiguous, of the context dtype, with %d elements" % (ncomp * self.N))
        return c_void_p(a.ctypes.data), HYDRO_MEM_HOST, a

    def load(self, T, pi=None):
        pT, mT, kT = self._ptr(T, 4)
        pP, mP, kP = self._ptr(pi, 10)
        if pi is not None and mP != mT:
            raise HydroError("T and pi must live in the same memory space")
        with self._torch.cuda.device(self.device):
            _check(self._lib.hydro_load(self._h, pT, pP, mT), "hydro_load")

    def set_history(self, u_prev):
        p, m, k = self._ptr(u_prev, 3)
        with self._torch.cuda.device(self.device):
            _check(self._lib.hydro_set_history(self._h, p, m), "hydro_set_history")

    def read_history(self, host=True):
        out = self._empty((3,) + self.shape, host)
        p, m, k = self._ptr(out, 3, writable=True)
        with self._torch.cuda.device(self.device):
            _check(self._lib.hydro_read_history(self._h, p, m), "hydro_read_history")
        return out

    def step(self, n=1):
        with self._torch.cuda.device(self.device):
            _check(self._lib.hydro_step(self._h, int(n)), "hydro_step")

    # -- eta_s-slab decomposition (hydro_stage / hydro_planes; paper_1802_04449_b200/slabs.py) ----------------
    def stage(self, which):
        """One stage of the current RK2 step: stage(1) then stage(2) is step(1)."""
        with self._torch.cuda.device(self.device):
            _check(self._lib.hydro_stage(self._h, int(which)), "hydro_stage")

    def plane_bytes(self) -> int:
        return int(self._lib.hydro_plane_bytes(self._h))

    def planes_get(self, which, k0, nk, host=False):
        """nk whole eta_s planes of a state buffer (0: current state, 1: stage-1 state) as opaque bytes (uint8 tensor)."""
        torch = self._torch
        n = nk * self.plane_bytes()
        buf = torch.empty(n, dtype=torch.uint8, device="cpu" if host else self.device)
        with torch.cuda.device(self.device):
            _check(self._lib.hydro_planes(self._h, int(which), int(k0), int(nk), c_void_p(buf.data_ptr()), 0,
                                          HYDRO_MEM_HOST if host else HYDRO_MEM_DEVICE), "hydro_planes")
        return buf

    def planes_put(self, which, k0, buf):
        """Write planes obtained from planes_get of a context with the same nx, ny, precision and viscosity."""
        nk, rem = divmod(buf.numel(), self.plane_bytes())
        if rem or buf.dtype != self._torch.uint8 or not buf.is_contiguous():
            raise HydroError("planes_put: a contiguous uint8 tensor of whole planes is required")
        with self._torch.cuda.device(self.device):
            _check(self._lib.hydro_planes(self._h, int(which), int(k0), int(nk), c_void_p(buf.data_ptr()), 1,
                                          HYDRO_MEM_DEVICE if buf.is_cuda else HYDRO_MEM_HOST), "hydro_planes")

    def _empty(self, shape, host, pinned=False):
        torch = self._torch
        if host:
            return torch.empty(shape, dtype=self.dtype, pin_memory=pinned).numpy() if not pinned else \
                torch.empty(shape, dtype=self.dtype, pin_memory=True)
        return torch.empty(shape, dtype=self.dtype, device=self.device)

    def read(self, host=True, out=None, want_pi=True):
        """Returns (e [nz,ny,nx], u [4,...], pi [10,...]); host=True -> numpy arrays, else CUDA tensors.
        out: optional (e, u, pi) buffers to fill (tensors or arrays in one memory space)."""
        if out is None:
            e = self._empty(self.shape, host)
            u = self._empty((4,) + self.shape, host)
            pi = self._empty((10,) + self.shape, host) if want_pi else None
        else:
            e, u, pi = out
        pe, me, _ = self._ptr(e, 1, writable=True)
        pu, mu, _ = self._ptr(u, 4, writable=True)
        pp, mp, _ = self._ptr(pi, 10, writable=True)
        with self._torch.cuda.device(self.device):
            _check(self._lib.hydro_read(self._h, pe, pu, pp, me), "hydro_read")
        return e, u, pi

    def diag(self):
        d = hydro_diag_t()
        with self._torch.cuda.device(self.device):
            warn = _check(self._lib.hydro_diag(self._h, byref(d)), "hydro_diag")
        return dict(tau=d.tau, step=int(d.step), cfl=tuple(d.cfl), e_max=d.e_max, floored=int(d.n_floor),
                    clamped=int(d.n_clamp), pi_limited=int(d.n_pi_limited), nan=int(d.n_nan),
                    root_unconverged=int(d.n_root_unconverged), warn=warn)

    # -- bulk pressure and net-baryon density (contexts created with bulk_baryon=1) ---------
    def load_ext(self, T, pi=None, Pi=None, nb=None):
        """hydro_load_ext: T^{tau mu} [4,...] (full tensor incl. Pi), pi [10,...], Pi [...], n [...]; all in one memory space."""
        pT, mT, k1 = self._ptr(T, 4)
        pp, mp, k2 = self._ptr(pi, 10)
        pP, mP, k3 = self._ptr(Pi, 1)
        pn, mn, k4 = self._ptr(nb, 1)
        with self._torch.cuda.device(self.device):
            _check(self._lib.hydro_load_ext(self._h, pT, pp, pP, pn, mT), "hydro_load_ext")

    def read_ext(self, host=True):
        """(Pi, n) of the current state, each [nz, ny, nx]."""
        Pi, nb = self._empty(self.shape, host), self._empty(self.shape, host)
        pP, mP, _ = self._ptr(Pi, 1, writable=True)
        pn, mn, _ = self._ptr(nb, 1, writable=True)
        with self._torch.cuda.device(self.device):
            _check(self._lib.hydro_read_ext(self._h, pP, pn, mP), "hydro_read_ext")
        return Pi, nb

    # -- freeze-out hypersurface -------------------------------------------------
    def freezeout_begin(self, e_frz, capacity):
        """Store the current state as level a; allocate the finder's workspace and the element arrays (device)."""
        torch = self._torch
        with torch.cuda.device(self.device):
            nbytes = int(self._lib.hydro_freezeout_bytes(byref(self.grid), self.precision))
            self._frz_ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = (self._frz_ws.data_ptr() + 255) // 256 * 256
            self._frz_keys = torch.empty(capacity, dtype=torch.int64, device=self.device)
            self._frz_rows = torch.empty((capacity, 22), dtype=torch.float64, device=self.device)
            self._frz_cap, self._frz_n = int(capacity), 0
            _check(self._lib.hydro_freezeout_begin(self._h, c_void_p(base), nbytes, float(e_frz)),
                   "hydro_freezeout_begin")

    def freezeout_slab(self):
        """Append the elements between the stored level and the current state; returns (n_total, n_hot)."""
        n, hot = c_longlong(0), c_longlong(0)
        with self._torch.cuda.device(self.device):
            _check(self._lib.hydro_freezeout_slab(self._h, c_void_p(self._frz_keys.data_ptr()),
                                                  c_void_p(self._frz_rows.data_ptr()), self._frz_cap, byref(n),
                                                  byref(hot)), "hydro_freezeout_slab")
        self._frz_n = int(n.value)
        return self._frz_n, int(hot.value)

    def freezeout_run(self, steps_per_slab, max_slabs):
        """{step(steps_per_slab); slab} until no cell is hotter than e_frz or max_slabs; returns
        (n_total, slabs done)."""
        n, ns = c_longlong(0), c_int(0)
        with self._torch.cuda.device(self.device):
            _check(self._lib.hydro_freezeout_run(self._h, int(steps_per_slab), int(max_slabs),
                                                 c_void_p(self._frz_keys.data_ptr()),
                                                 c_void_p(self._frz_rows.data_ptr()), self._frz_cap, byref(n),
                                                 byref(ns)), "hydro_freezeout_run")
        self._frz_n = int(n.value)
        return self._frz_n, int(ns.value)

    def freezeout_elements(self):
        """(keys int64 [M], rows float64 [M, 22]) gathered so far, as CUDA tensors in emission order."""
        return self._frz_keys[:self._frz_n], self._frz_rows[:self._frz_n]

    def launch_count(self) -> int:
        return int(self._lib.hydro_launch_count(self._h))

    def kernel(self) -> int:
        """The stage kernel in use (1 reference, 2 per-cell fused, 3 tile, 4 marching per-cell); kernel=0 resolves to the
        fastest measured (4 from 5e5 cells on, else 2)."""
        return int(self._lib.hydro_kernel(self._h))

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self._lib.hydro_destroy(self._h)
            self._h = c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def from_config(cfg, eos, **kw):
    """Hydro for an inputs.Config."""
    return Hydro(cfg.nx, cfg.ny, cfg.nz, cfg.dx, cfg.dy, cfg.deta, cfg.dtau, cfg.tau0, eos, cfg.eta_over_s,
                 bc=cfg.bc, geometry=cfg.geometry, **kw)

"""Thin ctypes binding of libclt.so (include/clt.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of ``csrc/``; torch is used for device memory
(the workspace tensor) and streams.  There is no CPU fallback: if ``libclt.so`` is missing or cannot
be loaded, importing/using this module raises.  Never imports ``oracle``.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libclt.so")

CLT_OK, CLT_EINVAL, CLT_ENOMEM, CLT_ESTATE, CLT_ECUDA, CLT_ENONFINITE = 0, -1, -2, -3, -4, -5


class clt_grid(ctypes.Structure):
    _fields_ = [("nR", ctypes.c_int32), ("nphi", ctypes.c_int32), ("nZ", ctypes.c_int32),
                ("Rmin", ctypes.c_double), ("Rmax", ctypes.c_double), ("Zmin", ctypes.c_double),
                ("Zmax", ctypes.c_double), ("phi_extent", ctypes.c_double)]


class clt_params(ctypes.Structure):
    _fields_ = [("gamma", ctypes.c_double), ("eta", ctypes.c_double), ("nu", ctypes.c_double),
                ("D", ctypes.c_double), ("kappa", ctypes.c_double), ("dt", ctypes.c_double),
                ("cfl", ctypes.c_double), ("flags", ctypes.c_uint32), ("d_i", ctypes.c_double)]


class clt_diag(ctypes.Structure):
    _fields_ = [("kinetic", ctypes.c_double), ("magnetic", ctypes.c_double), ("magnetic_pert", ctypes.c_double),
                ("magnetic_n1", ctypes.c_double), ("max_divB", ctypes.c_double), ("step", ctypes.c_int64),
                ("time", ctypes.c_double)]


class clt_profile(ctypes.Structure):
    _fields_ = [("ms_curl", ctypes.c_double), ("n_curl", ctypes.c_int64), ("ms_rhs", ctypes.c_double * 5),
                ("n_rhs", ctypes.c_int64 * 5), ("dropped", ctypes.c_int64), ("ms_phi", ctypes.c_double),
                ("n_phi", ctypes.c_int64)]


# every symbol include/clt.h declares
EXPORTS = ["clt_workspace_bytes", "clt_create", "clt_destroy", "clt_set_equilibrium", "clt_set_state", "clt_get_state",
           "clt_rhs", "clt_curl_J1", "clt_hall_G", "clt_step", "clt_step_cfl", "clt_step_stage", "clt_get_rows", "clt_set_rows",
           "clt_set_owned_rows", "clt_diagnostics_static", "clt_set_z_spacing", "clt_push_rows", "clt_link_rows", "clt_sync_peers", "clt_cfl_open", "clt_cfl_commit", "clt_cfl_close", "clt_set_dt", "clt_diagnostics", "clt_suggest_dt", "clt_set_tuning",
           "clt_set_kernel_variant", "clt_spectral_workspace_bytes", "clt_set_phi_scheme", "clt_set_profiling", "clt_get_profile", "clt_launch_count", "clt_stream", "clt_strerror", "clt_last_cuda_error", "clt_version"]

LIB_TEXTBOOK_PATH = os.path.join(_HERE, "libclt_textbook.so")
_lib = None
_libs = {}


class CltError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libclt error {code}: {msg}")
        self.code = code


def load(path=None):
    """Loads libclt.so (loudly).  Building is a separate, explicit step: ``python -m paper_1812_00525_b200.build``.
    ``path`` selects another build of the same ABI (libclt_textbook.so, the textbook-RK4-schedule A/B)."""
    global _lib
    path = path or LIB_PATH
    if path in _libs:
        return _libs[path]
    if not os.path.exists(path):
        raise ImportError(f"{path} not found: build it with `python -m paper_1812_00525_b200.build` "
                          "(there is no CPU fallback)")
    L = ctypes.CDLL(path)
    vp, i, d = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    L.clt_workspace_bytes.restype = ctypes.c_size_t
    L.clt_workspace_bytes.argtypes = [ctypes.POINTER(clt_grid)]
    L.clt_create.restype = i
    L.clt_create.argtypes = [ctypes.POINTER(clt_grid), ctypes.POINTER(clt_params), vp, ctypes.c_size_t, vp,
                             ctypes.POINTER(vp)]
    for name in ("clt_destroy",):
        getattr(L, name).restype = i
        getattr(L, name).argtypes = [vp]
    for name in ("clt_set_equilibrium", "clt_set_state", "clt_get_state", "clt_rhs", "clt_curl_J1", "clt_hall_G"):
        getattr(L, name).restype = i
        getattr(L, name).argtypes = [vp, vp]
    L.clt_step.restype = i
    L.clt_step.argtypes = [vp, i]
    L.clt_set_dt.restype = i
    L.clt_set_dt.argtypes = [vp, d]
    L.clt_diagnostics.restype = i
    L.clt_diagnostics.argtypes = [vp, ctypes.POINTER(clt_diag)]
    L.clt_diagnostics_static.restype = i
    L.clt_diagnostics_static.argtypes = [vp, d, vp]
    L.clt_suggest_dt.restype = i
    L.clt_suggest_dt.argtypes = [vp, d, ctypes.POINTER(d)]
    L.clt_set_tuning.restype = i
    L.clt_set_tuning.argtypes = [vp, i, i, i]
    L.clt_set_kernel_variant.restype = i
    L.clt_set_kernel_variant.argtypes = [vp, i]
    L.clt_set_profiling.restype = i
    L.clt_set_profiling.argtypes = [vp, i]
    L.clt_get_profile.restype = i
    L.clt_get_profile.argtypes = [vp, ctypes.POINTER(clt_profile)]
    L.clt_step_cfl.restype = i
    L.clt_step_cfl.argtypes = [vp, i, d, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    L.clt_step_stage.restype = i
    L.clt_step_stage.argtypes = [vp, i]
    for name in ("clt_get_rows", "clt_set_rows"):
        getattr(L, name).restype = i
        getattr(L, name).argtypes = [vp, i, i, i, vp]
    L.clt_set_owned_rows.restype = i
    L.clt_set_owned_rows.argtypes = [vp, i, i, i, i]
    L.clt_link_rows.restype = i
    L.clt_link_rows.argtypes = [vp, i, vp, i, i, i]
    L.clt_sync_peers.restype = i
    L.clt_sync_peers.argtypes = [vp, vp]
    L.clt_cfl_open.restype = i
    L.clt_cfl_open.argtypes = [vp, d]
    L.clt_cfl_commit.restype = i
    L.clt_cfl_commit.argtypes = [ctypes.POINTER(vp), i, i]
    L.clt_cfl_close.restype = i
    L.clt_cfl_close.argtypes = [vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    L.clt_set_z_spacing.restype = i
    L.clt_set_z_spacing.argtypes = [vp, d]
    L.clt_push_rows.restype = i
    L.clt_push_rows.argtypes = [vp, i, i, i, vp, i]
    L.clt_spectral_workspace_bytes.restype = ctypes.c_size_t
    L.clt_spectral_workspace_bytes.argtypes = [ctypes.POINTER(clt_grid)]
    L.clt_set_phi_scheme.restype = i
    L.clt_set_phi_scheme.argtypes = [vp, i, vp, ctypes.c_size_t]
    L.clt_launch_count.restype = ctypes.c_int64
    L.clt_launch_count.argtypes = [vp]
    L.clt_stream.restype = vp
    L.clt_stream.argtypes = [vp]
    L.clt_strerror.restype = ctypes.c_char_p
    L.clt_strerror.argtypes = [i]
    L.clt_last_cuda_error.restype = ctypes.c_char_p
    L.clt_last_cuda_error.argtypes = [vp]
    L.clt_version.restype = ctypes.c_char_p
    L.clt_version.argtypes = []
    _libs[path] = L
    if path == LIB_PATH:
        _lib = L
    return L


def _addr(a):
    """Address of a buffer: torch tensor (host or device), numpy array, or None."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        if a.dtype != np.float64 or not a.flags["C_CONTIGUOUS"]:
            raise TypeError("numpy buffers must be C-contiguous float64")
        return a.ctypes.data
    import torch
    if isinstance(a, torch.Tensor):
        if a.dtype != torch.float64 or not a.is_contiguous():
            raise TypeError("torch buffers must be contiguous float64")
        return a.data_ptr()
    raise TypeError(type(a))


class Clt:
    """One libclt context.  Method names and semantics are those of include/clt.h."""

    def __init__(self, nR, nphi, nZ, Rmin, Rmax, Zmin, Zmax, phi_extent=0.0, gamma=5.0 / 3.0, eta=0.0, nu=0.0, D=0.0,
                 kappa=0.0, dt=0.0, cfl=0.5, d_i=0.0, device="cuda:0", stream=None, lib_path=None):
        import torch
        self.L = load(lib_path)
        if not torch.cuda.is_available():
            raise RuntimeError("libclt needs a CUDA device (no CPU fallback)")
        self.device = torch.device(device)
        self.grid = clt_grid(nR, nphi, nZ, Rmin, Rmax, Zmin, Zmax, phi_extent)
        self.params = clt_params(gamma, eta, nu, D, kappa, dt, cfl, 0, d_i)
        self.shape = (8, nphi, nZ, nR)
        nbytes = self.L.clt_workspace_bytes(ctypes.byref(self.grid))
        if nbytes == 0:
            raise CltError(CLT_EINVAL, "invalid grid")
        self.workspace_bytes = nbytes
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)   # caching allocator: 512-B aligned
            self.torch_stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = ctypes.c_void_p()
            rc = self.L.clt_create(ctypes.byref(self.grid), ctypes.byref(self.params), self.workspace.data_ptr(), nbytes,
                                   ctypes.c_void_p(self.torch_stream.cuda_stream), ctypes.byref(h))
        self.h = h
        if rc != 0:
            self.h = None
            raise CltError(rc, self.L.clt_strerror(rc).decode())

    @classmethod
    def from_config(cls, cfg, dt, **kw):
        return cls(cfg.nR, cfg.nphi, cfg.nZ, cfg.Rmin, cfg.Rmax, cfg.Zmin, cfg.Zmax, cfg.phi_extent, cfg.gamma, cfg.eta,
                   cfg.nu, cfg.D, cfg.kappa, dt, cfg.cfl, **kw)

    def _ck(self, rc):
        if rc != 0:
            msg = self.L.clt_strerror(rc).decode()
            if rc == CLT_ECUDA and self.h:
                msg += " -- " + self.L.clt_last_cuda_error(self.h).decode()
            raise CltError(rc, msg)

    def close(self):
        if getattr(self, "h", None):
            self.L.clt_destroy(self.h)
            self.h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_equilibrium(self, U0):
        self._ck(self.L.clt_set_equilibrium(self.h, _addr(U0)))

    def set_state(self, U):
        self._ck(self.L.clt_set_state(self.h, _addr(U)))

    def get_state(self, out=None):
        if out is None:
            out = np.empty(self.shape)
        self._ck(self.L.clt_get_state(self.h, _addr(out)))
        return out

    def rhs(self, out=None):
        if out is None:
            out = np.empty(self.shape)
        self._ck(self.L.clt_rhs(self.h, _addr(out)))
        return out

    def curl_J1(self, out=None):
        if out is None:
            out = np.empty((3,) + self.shape[1:])
        self._ck(self.L.clt_curl_J1(self.h, _addr(out)))
        return out

    def step_cfl(self, n, cfl=0.0):
        """n adaptive RK4 steps (dt = SETDT per step, on the device); returns (dt of the next step, time advanced)."""
        a, b = ctypes.c_double(), ctypes.c_double()
        self._ck(self.L.clt_step_cfl(self.h, int(n), float(cfl), ctypes.byref(a), ctypes.byref(b)))
        return a.value, b.value

    def step_stage(self, stage):
        self._ck(self.L.clt_step_stage(self.h, int(stage)))

    def get_rows(self, buffer, k0, nrows, out):
        """out: numpy array or torch tensor (host or device), float64, dense [8][nphi][nrows][nR]."""
        self._ck(self.L.clt_get_rows(self.h, int(buffer), int(k0), int(nrows), _addr(out)))
        return out

    def set_rows(self, buffer, k0, nrows, src):
        self._ck(self.L.clt_set_rows(self.h, int(buffer), int(k0), int(nrows), _addr(src)))

    def set_owned_rows(self, k_first, k_last, deep_first, deep_last):
        self._ck(self.L.clt_set_owned_rows(self.h, int(k_first), int(k_last), int(deep_first), int(deep_last)))

    def cfl_open(self, cfl=0.0):
        self._ck(self.L.clt_cfl_open(self.h, float(cfl)))

    def cfl_close(self):
        """Returns (dt of the next step, time advanced since cfl_open)."""
        a, b = ctypes.c_double(), ctypes.c_double()
        self._ck(self.L.clt_cfl_close(self.h, ctypes.byref(a), ctypes.byref(b)))
        return a.value, b.value

    def set_z_spacing(self, dZ):
        """A slab of a larger grid: the global dZ, bit for bit (call before set_equilibrium / set_state)."""
        self._ck(self.L.clt_set_z_spacing(self.h, float(dZ)))

    def push_rows(self, buffer, k0, nrows, dst, k0_dst):
        """Rows k0 .. k0+nrows-1 of `buffer` of this context -> rows k0_dst .. of the same buffer of context `dst`."""
        rc = self.L.clt_push_rows(self.h, int(buffer), int(k0), int(nrows), dst.h, int(k0_dst))
        if rc != 0:
            dst._ck(rc)

    def link_rows(self, side, peer, k0=0, nrows=0, k0_peer=0):
        """Every stage kernel also stores rows k0 .. k0+nrows-1 of its output into rows k0_peer .. of `peer` (None: unlink)."""
        self._ck(self.L.clt_link_rows(self.h, int(side), peer.h if peer is not None else None, int(k0), int(nrows), int(k0_peer)))

    def sync_peers(self, other):
        self._ck(self.L.clt_sync_peers(self.h, other.h))

    def hall_G(self, out=None):
        if out is None:
            out = np.empty((3,) + self.shape[1:])
        self._ck(self.L.clt_hall_G(self.h, _addr(out)))
        return out

    def step(self, n=1):
        self._ck(self.L.clt_step(self.h, int(n)))

    def set_dt(self, dt):
        self._ck(self.L.clt_set_dt(self.h, float(dt)))

    def diagnostics(self):
        d = clt_diag()
        self._ck(self.L.clt_diagnostics(self.h, ctypes.byref(d)))
        return {k: getattr(d, k) for k, _ in clt_diag._fields_}

    def diagnostics_static(self, out, cfl=0.0):
        """clt_diagnostics_static: the reductions with the library's static scratch (no allocation, no synchronisation).
        out: CUDA tensor of >= 6 float64: kinetic, magnetic, magnetic_pert, magnetic_n1, max_divB, SETDT(cfl)."""
        self._ck(self.L.clt_diagnostics_static(self.h, float(cfl), _addr(out)))
        return out

    def suggest_dt(self, cfl=0.0):
        out = ctypes.c_double()
        self._ck(self.L.clt_suggest_dt(self.h, float(cfl), ctypes.byref(out)))
        return out.value

    def set_tuning(self, tile_z=0, phi_chunks=0, use_graph=0):
        self._ck(self.L.clt_set_tuning(self.h, int(tile_z), int(phi_chunks), int(use_graph)))

    def set_kernel_variant(self, variant=0):
        self._ck(self.L.clt_set_kernel_variant(self.h, int(variant)))

    def set_phi_scheme(self, scheme=1):
        """0 = 4th-order finite differences in phi (default), 1 = pseudo-spectral (allocates the scratch tensor)."""
        import torch
        if not scheme:
            self._ck(self.L.clt_set_phi_scheme(self.h, 0, None, 0))
            self._spec_ws = None
            return
        nbytes = self.L.clt_spectral_workspace_bytes(ctypes.byref(self.grid))
        if nbytes == 0:
            raise CltError(CLT_EINVAL, "pseudo-spectral scheme: nphi too large")
        ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        off = (-ws.data_ptr()) % 256
        self._ck(self.L.clt_set_phi_scheme(self.h, int(scheme), ws.data_ptr() + off, nbytes))
        self._spec_ws = ws

    def set_profiling(self, enable=True):
        self._ck(self.L.clt_set_profiling(self.h, int(bool(enable))))

    def get_profile(self):
        p = clt_profile()
        self._ck(self.L.clt_get_profile(self.h, ctypes.byref(p)))
        return {"ms_curl": p.ms_curl, "n_curl": p.n_curl, "ms_rhs": list(p.ms_rhs), "n_rhs": list(p.n_rhs),
                "dropped": p.dropped, "ms_phi": p.ms_phi, "n_phi": p.n_phi}

    @property
    def launch_count(self):
        return int(self.L.clt_launch_count(self.h))


def cfl_commit(ctxs, init):
    """clt_cfl_commit over the contexts `ctxs` (Clt objects of one library build and one device)."""
    arr = (ctypes.c_void_p * len(ctxs))(*[c.h for c in ctxs])
    ctxs[0]._ck(ctxs[0].L.clt_cfl_commit(arr, len(ctxs), int(bool(init))))


def version():
    return load().clt_version().decode()

"""Thin Python binding of the C-ABI in include/f4.h (same call names).

Argument marshalling only: every step of the path runs in the CUDA kernels of
``libf4.so``.  PyTorch supplies device memory (the block store) and the
stream; numpy supplies host buffers.  There is no CPU fallback: device calls
raise ``F4Error`` when the library or a CUDA device is missing.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

F4_OK = 0
ERRORS = {-1: "F4_EINVAL", -2: "F4_ENOBLOCKS", -3: "F4_ECUDA", -4: "F4_EUNBOUND", -5: "F4_EUNBALANCED",
          -6: "F4_EUNSUPPORTED"}
BC_PERIODIC, BC_OUTFLOW, BC_KEEP, BC_DIRICHLET, BC_NEUMANN, BC_DATA = 0, 1, 2, 3, 4, 5
BC_DATA_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_double))
LIM_VANLEER, LIM_MINMOD, LIM_MC, LIM_KOREN, LIM_WENO3 = 0, 1, 2, 3, 4
FLUX_HLL, FLUX_RUSANOV = 0, 1
CRIT_LOHNER, CRIT_PJUMP = 0, 1
RK_HEUN, RK_EULER, RK_SSP33, RK_SSP43, RK_RK4 = 0, 1, 2, 3, 4
RK_STAGES = {RK_HEUN: 2, RK_EULER: 1, RK_SSP33: 3, RK_SSP43: 4, RK_RK4: 4}
RK_STATES = {RK_HEUN: 2, RK_EULER: 2, RK_SSP33: 3, RK_SSP43: 3, RK_RK4: 4}
OP_SRL, OP_BC, OP_F2C, OP_C2F = 0, 1, 2, 3
PROF_NAMES = ("ghost_r1", "ghost_r2", "stage", "dt_reduce", "regrid", "layout")

# every symbol include/f4.h declares
SYMBOLS = ("f4_mesh_create", "f4_mesh_destroy", "f4_set_options", "f4_set_flux_fix", "f4_set_physics", "f4_num_vars", "f4_set_bc_values", "f4_set_bc_callback", "f4_update_bc_data",
           "f4_num_bc_faces", "f4_set_gravity", "f4_set_rk_scheme", "f4_storage_bytes", "f4_bind_storage",
           "f4_num_blocks", "f4_get_blocks", "f4_set_state", "f4_get_state", "f4_build_ghost_pattern",
           "f4_pattern_size", "f4_get_pattern", "f4_fill_ghosts", "f4_compute_dt", "f4_advance", "f4_advance_cfl", "f4_last_dt", "f4_refine_flags", "f4_adapt", "f4_adapt_begin", "f4_adapt_end",
           "f4_conserved_totals", "f4_conserved_totals_noalloc", "f4_profile_enable", "f4_profile_get", "f4_launch_count", "f4_last_adapt_ms", "f4_last_error",
           "f4_version")


PHYS_EULER, PHYS_ADVECTION = 0, 1
NOALLOC_MAX_BLOCKS = 32768   # F4_NOALLOC_MAX_BLOCKS


class F4Error(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{ERRORS.get(code, code)}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load libf4.so (built in-tree by build.py; fails loudly if it cannot be built or loaded)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if not os.path.exists(path):
        path = _build.build()
    L = C.CDLL(path)
    vp, ip, dp = C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_double)
    L.f4_mesh_create.argtypes = [C.c_int, C.c_int, C.c_int, ip, C.c_int, C.c_int, ip, C.c_double, C.c_int, C.c_int,
                                 C.POINTER(vp)]
    L.f4_mesh_destroy.argtypes = [vp]
    L.f4_set_options.argtypes = [vp, C.c_int, C.c_int, C.c_double]
    L.f4_set_flux_fix.argtypes = [vp, C.c_int]
    L.f4_set_physics.argtypes = [vp, C.c_int, dp]
    L.f4_num_vars.argtypes = [vp]
    L.f4_set_rk_scheme.argtypes = [vp, C.c_int]
    L.f4_set_gravity.argtypes = [vp, dp]
    L.f4_set_bc_values.argtypes = [vp, dp]
    L.f4_set_bc_callback.argtypes = [vp, BC_DATA_FN, vp]
    L.f4_update_bc_data.argtypes = [vp]
    L.f4_num_bc_faces.argtypes = [vp]
    L.f4_refine_flags.argtypes = [vp, C.c_int, C.c_int, C.c_int, dp, ip, dp]
    L.f4_storage_bytes.restype = C.c_size_t
    L.f4_storage_bytes.argtypes = [vp]
    L.f4_bind_storage.argtypes = [vp, vp, C.c_size_t, vp]
    L.f4_num_blocks.argtypes = [vp]
    L.f4_get_blocks.argtypes = [vp, ip, ip, dp, dp]
    L.f4_set_state.argtypes = [vp, C.c_int, vp, C.c_int, C.c_int]
    L.f4_get_state.argtypes = [vp, C.c_int, vp, C.c_int, C.c_int]
    L.f4_build_ghost_pattern.argtypes = [vp]
    L.f4_pattern_size.argtypes = [vp, ip, ip]
    L.f4_get_pattern.argtypes = [vp, ip]
    L.f4_fill_ghosts.argtypes = [vp, C.c_int]
    L.f4_compute_dt.argtypes = [vp, C.c_int, C.c_double, dp]
    L.f4_advance.argtypes = [vp, C.c_double]
    L.f4_adapt.argtypes = [vp, ip, ip]
    L.f4_advance_cfl.argtypes = [vp, C.c_double]
    L.f4_last_dt.argtypes = [vp, dp]
    L.f4_adapt_begin.argtypes = [vp, ip]
    L.f4_adapt_end.argtypes = [vp, ip]
    L.f4_conserved_totals.argtypes = [vp, C.c_int, dp]
    L.f4_conserved_totals_noalloc.argtypes = [vp, C.c_int, vp]
    L.f4_profile_enable.argtypes = [vp, C.c_int]
    L.f4_profile_get.argtypes = [vp, dp, C.POINTER(C.c_longlong), C.c_int]
    L.f4_launch_count.restype = C.c_longlong
    L.f4_launch_count.argtypes = [vp]
    L.f4_last_adapt_ms.argtypes = [vp, dp]
    L.f4_last_error.restype = C.c_char_p
    L.f4_last_error.argtypes = [vp]
    L.f4_version.restype = C.c_char_p
    _lib = L
    return L


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class Mesh:
    """Owner of an ``f4_mesh*`` and (optionally) of the torch tensor lent to it as block store."""

    def __init__(self, dim, block_n, n_ghost, brick, base_level, max_level, bc_kind, gamma=1.4, n_states=2,
                 max_blocks=None):
        self.L = lib()
        self.dim, self.N, self.Ng = dim, block_n, n_ghost
        self.P = block_n + 2 * n_ghost
        self.nvar = dim + 2
        self.gamma = gamma
        br = np.asarray(list(brick) + [1] * (3 - len(brick)), dtype=np.int32)
        bc = np.asarray(list(bc_kind) + [0] * (6 - len(bc_kind)), dtype=np.int32)
        if max_blocks is None:
            max_blocks = int(np.prod([int(br[a]) << base_level for a in range(dim)]))
        self.max_blocks = max_blocks
        h = C.c_void_p()
        rc = self.L.f4_mesh_create(dim, block_n, n_ghost, _ip(br), base_level, max_level, _ip(bc), gamma, n_states,
                                   max_blocks, C.byref(h))
        if rc != F4_OK:
            raise F4Error(rc, "f4_mesh_create")
        self.h = h
        self._store = None

    @classmethod
    def from_config(cls, cfg, n_states=2, max_blocks=None):
        if cfg.get("physics") == "advection":
            m = cls._from_config_base(cfg, n_states, max_blocks)
            m.set_advection(cfg["velocity"])
            return m
        return cls._from_config_base(cfg, n_states, max_blocks)

    @classmethod
    def _from_config_base(cls, cfg, n_states=2, max_blocks=None):
        return cls(cfg["dim"], cfg["block_n"], cfg["n_ghost"], cfg["brick"], cfg["base_level"], cfg["max_level"],
                   cfg["bc"], cfg["gamma"], n_states, max_blocks)

    def close(self):
        if getattr(self, "h", None):
            self.L.f4_mesh_destroy(self.h)
            self.h = None
            self._store = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, rc):
        if rc != F4_OK:
            raise F4Error(rc, self.L.f4_last_error(self.h).decode())

    # -- storage -----------------------------------------------------------
    def storage_bytes(self):
        return self.L.f4_storage_bytes(self.h)

    def bind_storage(self, dev_ptr, nbytes, stream=0):
        self._chk(self.L.f4_bind_storage(self.h, C.c_void_p(dev_ptr), nbytes, C.c_void_p(stream)))

    def bind_torch(self, device="cuda:0", stream=None):
        """Allocate the block store as a torch tensor on ``device`` and lend it to the mesh."""
        import torch
        if not torch.cuda.is_available():
            raise F4Error(-3, "no CUDA device: the f4 path has no CPU fallback")
        nbytes = self.storage_bytes()
        self._store = torch.empty(nbytes // 8, dtype=torch.float64, device=device)
        s = stream if stream is not None else torch.cuda.current_stream(device)
        self._stream = s
        self.bind_storage(self._store.data_ptr(), nbytes, s.cuda_stream)
        return self._store

    # -- mesh --------------------------------------------------------------
    @property
    def num_blocks(self):
        return self.L.f4_num_blocks(self.h)

    def get_blocks(self, geometry=False):
        nb = self.num_blocks
        lev = np.zeros(nb, dtype=np.int32)
        co = np.zeros((nb, 3), dtype=np.int32)
        if not geometry:
            self._chk(self.L.f4_get_blocks(self.h, _ip(lev), _ip(co), None, None))
            return lev, co
        org = np.zeros((nb, 3))
        dx = np.zeros(nb)
        self._chk(self.L.f4_get_blocks(self.h, _ip(lev), _ip(co), _dp(org), _dp(dx)))
        return lev, co, org, dx

    def set_options(self, limiter=LIM_VANLEER, flux=FLUX_HLL, theta=1.0):
        self._chk(self.L.f4_set_options(self.h, limiter, flux, theta))

    def set_bc_values(self, values):
        v = np.ascontiguousarray(values, dtype=np.float64)
        assert v.shape == (6, self.nvar)
        self._chk(self.L.f4_set_bc_values(self.h, _dp(v)))

    def set_bc_callback(self, fn):
        """fn(blocks[n], faces[n], out[n, nvar, kmax, N]) fills the boundary values of the F4_BC_DATA faces
        (eq. 4); the library calls it whenever the face list changes and on update_bc_data()."""
        nvar, N, kmax = self.nvar, self.N, (self.N if self.dim == 3 else 1)

        def tramp(_user, n, blk, face, data):
            b = np.ctypeslib.as_array(blk, shape=(n,)).copy()
            f = np.ctypeslib.as_array(face, shape=(n,)).copy()
            out = np.ctypeslib.as_array(data, shape=(n, nvar, kmax, N))
            fn(b, f, out)

        self._bc_cb = BC_DATA_FN(tramp)          # keep the trampoline alive as long as the mesh
        self._chk(self.L.f4_set_bc_callback(self.h, self._bc_cb, None))

    def update_bc_data(self):
        self._chk(self.L.f4_update_bc_data(self.h))

    @property
    def num_bc_faces(self):
        return self.L.f4_num_bc_faces(self.h)

    def set_advection(self, velocity):
        """Scalar advection eq. (13) with a uniform velocity field: one variable per cell.
        Before bind_storage / bind_torch."""
        v = np.zeros(3)
        v[:self.dim] = np.asarray(velocity, dtype=np.float64)[:self.dim]
        self._chk(self.L.f4_set_physics(self.h, PHYS_ADVECTION, _dp(v)))
        self.nvar = 1

    def set_gravity(self, g):
        gg = np.zeros(3, dtype=np.float64)
        gg[:len(g)] = g
        self._chk(self.L.f4_set_gravity(self.h, _dp(gg)))

    def set_rk_scheme(self, scheme):
        self._chk(self.L.f4_set_rk_scheme(self.h, int(scheme)))

    def set_flux_fix(self, on=True):
        self._chk(self.L.f4_set_flux_fix(self.h, int(on)))

    def build_ghost_pattern(self):
        self._chk(self.L.f4_build_ghost_pattern(self.h))

    def pattern(self):
        n1, n2 = C.c_int(), C.c_int()
        self._chk(self.L.f4_pattern_size(self.h, C.byref(n1), C.byref(n2)))
        rec = np.zeros((n1.value + n2.value, 6), dtype=np.int32)
        if rec.size:
            self._chk(self.L.f4_get_pattern(self.h, _ip(rec)))
        return rec, n1.value, n2.value

    def refine_flags(self, state, criterion, params, var=0):
        """(flags, indicator) per block, computed on the device (f4_refine_flags)."""
        pr = np.zeros(4, dtype=np.float64)
        pr[:len(params)] = params
        flags = np.zeros(self.num_blocks, dtype=np.int32)
        ind = np.zeros(self.num_blocks, dtype=np.float64)
        self._chk(self.L.f4_refine_flags(self.h, state, criterion, var, _dp(pr), _ip(flags), _dp(ind)))
        return flags, ind

    def adapt(self, flags):
        f = np.ascontiguousarray(flags, dtype=np.int32)
        assert f.shape[0] == self.num_blocks
        ch = C.c_int(0)
        self._chk(self.L.f4_adapt(self.h, _ip(f), C.byref(ch)))
        return bool(ch.value)

    def advance_cfl(self, cfl):
        """compute_dt + advance without a host round trip (dt stays on the device); last_dt() reads it back."""
        self._chk(self.L.f4_advance_cfl(self.h, float(cfl)))

    def last_dt(self):
        dt = C.c_double(0.0)
        self._chk(self.L.f4_last_dt(self.h, C.byref(dt)))
        return dt.value

    def adapt_begin(self, flags):
        """Start the host part of a regrid on a worker thread (compute_dt / advance may follow); adapt_end() commits."""
        f = np.ascontiguousarray(flags, dtype=np.int32)
        assert f.shape[0] == self.num_blocks
        self._chk(self.L.f4_adapt_begin(self.h, _ip(f)))

    def adapt_end(self):
        ch = C.c_int(0)
        self._chk(self.L.f4_adapt_end(self.h, C.byref(ch)))
        return bool(ch.value)

    # -- state -------------------------------------------------------------
    def _shape(self, with_ghosts):
        n = self.P if with_ghosts else self.N
        return (self.num_blocks, self.nvar, n if self.dim == 3 else 1, n, n)

    def set_state(self, state, arr, with_ghosts=False):
        """arr: numpy array (host) or torch CUDA tensor (device), [nb][nvar][k][j][i]."""
        if isinstance(arr, np.ndarray):
            a = np.ascontiguousarray(arr, dtype=np.float64)
            assert a.shape == self._shape(with_ghosts), (a.shape, self._shape(with_ghosts))
            self._chk(self.L.f4_set_state(self.h, state, C.c_void_p(a.ctypes.data), 0, int(with_ghosts)))
        else:
            assert arr.is_contiguous() and arr.numel() == int(np.prod(self._shape(with_ghosts)))
            self._chk(self.L.f4_set_state(self.h, state, C.c_void_p(arr.data_ptr()), int(arr.is_cuda), int(with_ghosts)))

    def get_state(self, state, with_ghosts=False, out=None):
        if out is None:
            out = np.zeros(self._shape(with_ghosts), dtype=np.float64)
        if isinstance(out, np.ndarray):
            self._chk(self.L.f4_get_state(self.h, state, C.c_void_p(out.ctypes.data), 0, int(with_ghosts)))
        else:
            self._chk(self.L.f4_get_state(self.h, state, C.c_void_p(out.data_ptr()), int(out.is_cuda), int(with_ghosts)))
        return out

    # -- the step ------------------------------------------------------------
    def fill_ghosts(self, state):
        self._chk(self.L.f4_fill_ghosts(self.h, state))

    def compute_dt(self, state, cfl):
        dt = C.c_double()
        self._chk(self.L.f4_compute_dt(self.h, state, cfl, C.byref(dt)))
        return dt.value

    def advance(self, dt):
        self._chk(self.L.f4_advance(self.h, dt))

    def conserved_totals(self, state):
        out = np.zeros(self.nvar)
        self._chk(self.L.f4_conserved_totals(self.h, state, _dp(out)))
        return out

    def conserved_totals_noalloc(self, state, out_dev_ptr):
        """f4_conserved_totals_noalloc: totals into DEVICE memory at out_dev_ptr ([nvar] doubles, e.g. tensor.data_ptr()),
        enqueued on the mesh's stream, no synchronisation, no allocation (at most NOALLOC_MAX_BLOCKS blocks)."""
        self._chk(self.L.f4_conserved_totals_noalloc(self.h, state, C.c_void_p(int(out_dev_ptr))))

    # -- measurement ---------------------------------------------------------
    def profile_enable(self, on=True):
        self._chk(self.L.f4_profile_enable(self.h, int(on)))

    def profile_get(self, reset=True):
        ms = np.zeros(len(PROF_NAMES))
        n = np.zeros(len(PROF_NAMES), dtype=np.int64)
        self._chk(self.L.f4_profile_get(self.h, _dp(ms), n.ctypes.data_as(C.POINTER(C.c_longlong)), int(reset)))
        return {k: (float(ms[q]), int(n[q])) for q, k in enumerate(PROF_NAMES)}

    def launch_count(self):
        return self.L.f4_launch_count(self.h)

    def last_adapt_ms(self):
        ms = np.zeros(3)
        self._chk(self.L.f4_last_adapt_ms(self.h, _dp(ms)))
        return {"host_mesh_pattern": float(ms[0]), "transfer": float(ms[1]), "upload": float(ms[2])}


def version():
    return lib().f4_version().decode()

"""ORACLE -- TEST INFRASTRUCTURE ONLY.

ctypes wrapper around ``oracle/f4_oracle.cpp`` (the plain single-threaded CPU
statement of the hot path; see that file's header for scope, readings and
pins).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this module.  It never
imports ``paper_2605_07612_b200``.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "f4_oracle.cpp")
_LIB = os.path.join(_HERE, "libf4oracle.so")

LIM_VANLEER, LIM_MINMOD, LIM_MC, LIM_KOREN, LIM_WENO3 = 0, 1, 2, 3, 4
FLUX_HLL, FLUX_RUSANOV = 0, 1
NB_BOUNDARY, NB_SAME, NB_COARSE, NB_FINE = 0, 1, 2, 3


def build(force: bool = False) -> str:
    """g++ -O2 -ffp-contract=off: no FMA contraction, no fast-math."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC", "-pthread",
                               "-o", _LIB, _SRC])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int)
        L.ora_create.restype = C.c_void_p
        L.ora_create.argtypes = [C.c_int, C.c_int, C.c_int, ip, C.c_int, C.c_int, ip, C.c_double, C.c_int]
        L.ora_destroy.argtypes = [C.c_void_p]
        L.ora_set_options.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double]
        L.ora_set_test_rhs.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.ora_set_flux_fix.argtypes = [C.c_void_p, C.c_int]
        L.ora_set_gravity.argtypes = [C.c_void_p, dp]
        L.ora_set_physics.argtypes = [C.c_void_p, C.c_int, dp]
        L.ora_set_bc_values.argtypes = [C.c_void_p, dp]
        L.ora_set_bc_face_data.argtypes = [C.c_void_p, C.c_int, C.c_int, dp]
        L.ora_clear_bc_data.argtypes = [C.c_void_p]
        L.ora_num_blocks.argtypes = [C.c_void_p]
        L.ora_get_blocks.argtypes = [C.c_void_p, ip, ip]
        L.ora_dx.restype = C.c_double
        L.ora_dx.argtypes = [C.c_void_p, C.c_int]
        L.ora_last_error.restype = C.c_char_p
        L.ora_last_error.argtypes = [C.c_void_p]
        L.ora_set_state.argtypes = [C.c_void_p, C.c_int, dp, C.c_int]
        L.ora_get_state.argtypes = [C.c_void_p, C.c_int, dp, C.c_int]
        L.ora_fill_ghosts.argtypes = [C.c_void_p, C.c_int]
        L.ora_max_wave_rate.restype = C.c_double
        L.ora_max_wave_rate.argtypes = [C.c_void_p, C.c_int]
        L.ora_compute_dt.restype = C.c_double
        L.ora_compute_dt.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.ora_advance.argtypes = [C.c_void_p, C.c_double]
        L.ora_advance_mt.argtypes = [C.c_void_p, C.c_double, C.c_int]
        L.ora_compute_dt_mt.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_int]
        L.ora_compute_dt_mt.restype = C.c_double
        L.ora_advance_rk.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.ora_forward_euler.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_int, dp, ip]
        L.ora_adapt.argtypes = [C.c_void_p, ip, ip]
        L.ora_refine_flags.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, dp, ip, dp]
        L.ora_totals.argtypes = [C.c_void_p, C.c_int, dp]
        L.ora_permute.argtypes = [C.c_void_p, ip]
        L.ora_face_table.argtypes = [C.c_void_p, ip, ip, ip]
        L.ora_minmod_G.restype = C.c_double
        L.ora_minmod_G.argtypes = [C.c_double] * 3
        L.ora_vanleer.restype = C.c_double
        L.ora_vanleer.argtypes = [C.c_double] * 2
        L.ora_koren.restype = C.c_double
        L.ora_koren.argtypes = [C.c_double] * 2
        L.ora_weno3.restype = C.c_double
        L.ora_weno3.argtypes = [C.c_double] * 2
        L.ora_riemann_flux.argtypes = [C.c_int, C.c_double, C.c_int, dp, dp, C.c_int, dp]
        L.ora_to_primitive.argtypes = [C.c_int, C.c_double, dp, dp]
        L.ora_to_conservative.argtypes = [C.c_int, C.c_double, dp, dp]
        L.ora_advection_flux.argtypes = [C.c_int, dp, C.c_int, C.c_double, C.c_double, C.c_int]
        L.ora_advection_flux.restype = C.c_double
        L.ora_wavespeeds.argtypes = [C.c_int, C.c_double, dp, dp, C.c_int, dp, dp]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


class OracleError(RuntimeError):
    pass


class OracleMesh:
    """Mesh + block store of the oracle.  Same call names as the C-ABI of include/f4.h."""

    def __init__(self, dim, block_n, n_ghost, brick, base_level, max_level, bc_kind, gamma, n_states=2):
        self.L = lib()
        self.dim, self.N, self.Ng = dim, block_n, n_ghost
        self.P = block_n + 2 * n_ghost
        self.nvar = dim + 2
        self.gamma = gamma
        br = np.asarray(list(brick) + [1] * (3 - len(brick)), dtype=np.int32)
        bc = np.asarray(list(bc_kind) + [0] * (6 - len(bc_kind)), dtype=np.int32)
        self.h = self.L.ora_create(dim, block_n, n_ghost, _ip(br), base_level, max_level, _ip(bc), gamma, n_states)
        if not self.h:
            raise OracleError("ora_create: bad arguments")

    @classmethod
    def from_config(cls, cfg, n_states=2):
        m = cls(cfg["dim"], cfg["block_n"], cfg["n_ghost"], cfg["brick"], cfg["base_level"],
                cfg["max_level"], cfg["bc"], cfg["gamma"], n_states)
        if cfg.get("physics") == "advection":
            m.set_advection(cfg["velocity"])
        return m

    def set_advection(self, velocity):
        """Scalar advection eq. (13) with a uniform velocity field: one variable per cell.  Call
        before any state is set."""
        v = np.zeros(3)
        v[:self.dim] = np.asarray(velocity, dtype=np.float64)[:self.dim]
        self._chk(self.L.ora_set_physics(self.h, 1, _dp(v)))
        self.nvar = 1

    def __del__(self):
        if getattr(self, "h", None):
            self.L.ora_destroy(self.h)
            self.h = None

    def _chk(self, rc):
        if rc != 0:
            raise OracleError(self.L.ora_last_error(self.h).decode())

    def set_options(self, limiter=LIM_VANLEER, flux=FLUX_HLL, theta=1.0):
        self.L.ora_set_options(self.h, limiter, flux, theta)

    def set_bc_values(self, values):
        """values[6][nvar]: u_b of Dirichlet faces / normal derivative u_b' of Neumann faces."""
        v = np.ascontiguousarray(values, dtype=np.float64)
        assert v.shape == (6, self.nvar)
        self.L.ora_set_bc_values(self.h, _dp(v))

    def set_bc_data(self, faces, data):
        """Spatially varying boundary values (eq. 4) of the faces of kind 5 (BC_DATA):
        faces = [(block, face), ...], data[len(faces)][nvar][kmax][N].  Replaces all earlier data (the block
        numbering changes with the mesh)."""
        self.L.ora_clear_bc_data(self.h)
        d = np.ascontiguousarray(data, dtype=np.float64)
        for q, (b, f) in enumerate(faces):
            self.L.ora_set_bc_face_data(self.h, int(b), int(f), _dp(np.ascontiguousarray(d[q])))

    def set_gravity(self, g):
        """Gravitational acceleration of the source term eq. (20); (0,0,0) = no source."""
        gg = np.zeros(3, dtype=np.float64)
        gg[:len(g)] = g
        self.L.ora_set_gravity(self.h, _dp(gg))

    def set_flux_fix(self, on=True):
        """Conservative flux correction at refinement boundaries."""
        self.L.ora_set_flux_fix(self.h, int(on))

    def set_test_rhs(self, on, lam):
        self.L.ora_set_test_rhs(self.h, int(on), lam)

    @property
    def num_blocks(self):
        return self.L.ora_num_blocks(self.h)

    def get_blocks(self):
        nb = self.num_blocks
        lev = np.zeros(nb, dtype=np.int32)
        co = np.zeros((nb, 3), dtype=np.int32)
        self.L.ora_get_blocks(self.h, _ip(lev), _ip(co))
        return lev, co

    def dx(self, level):
        return self.L.ora_dx(self.h, int(level))

    def _shape(self, with_ghosts):
        n = self.P if with_ghosts else self.N
        nz = n if self.dim == 3 else 1
        return (self.num_blocks, self.nvar, nz, n, n)

    def set_state(self, state, arr, with_ghosts=False):
        a = np.ascontiguousarray(arr, dtype=np.float64)
        assert a.shape == self._shape(with_ghosts), (a.shape, self._shape(with_ghosts))
        self.L.ora_set_state(self.h, state, _dp(a), int(with_ghosts))

    def get_state(self, state, with_ghosts=False):
        out = np.zeros(self._shape(with_ghosts), dtype=np.float64)
        self.L.ora_get_state(self.h, state, _dp(out), int(with_ghosts))
        return out

    def fill_ghosts(self, state):
        self._chk(self.L.ora_fill_ghosts(self.h, state))

    def max_wave_rate(self, state):
        return self.L.ora_max_wave_rate(self.h, state)

    def compute_dt(self, state, cfl):
        return self.L.ora_compute_dt(self.h, state, cfl)

    RK_HEUN, RK_EULER, RK_SSP33, RK_SSP43, RK_RK4 = 0, 1, 2, 3, 4

    def advance(self, dt, scheme=None):
        """One step: Heun (eq. 6-7) by default, else the scheme of PAPER.md:296-314 (needs 3 / 4 states)."""
        if scheme is None:
            self._chk(self.L.ora_advance(self.h, dt))
        else:
            self._chk(self.L.ora_advance_rk(self.h, int(scheme), dt))

    def advance_mt(self, dt, nthreads):
        """Heun step by the block-parallel driver (timing only; bit-identical to advance)."""
        self._chk(self.L.ora_advance_mt(self.h, dt, int(nthreads)))

    def compute_dt_mt(self, state, cfl, nthreads):
        return self.L.ora_compute_dt_mt(self.h, state, cfl, int(nthreads))

    def forward_euler(self, s_out, s_deriv, dt_sub, w, s_prev):
        w = np.asarray(w, dtype=np.float64)
        sp = np.asarray(s_prev, dtype=np.int32)
        self._chk(self.L.ora_forward_euler(self.h, s_out, s_deriv, dt_sub, len(w), _dp(w), _ip(sp)))

    def adapt(self, flags):
        f = np.ascontiguousarray(flags, dtype=np.int32)
        assert f.shape[0] == self.num_blocks
        ch = C.c_int(0)
        self._chk(self.L.ora_adapt(self.h, _ip(f), C.byref(ch)))
        return bool(ch.value)

    CRIT_LOHNER, CRIT_PJUMP = 0, 1

    def refine_flags(self, state, criterion, params, var=0):
        """Per-block flags and indicator of a GHOST-FILLED state: criterion 0 = eq. (12) with
        params (c_refine, c_derefine, eps, eps_abs) on stored variable var; 1 = pressure jump (reading A15) with
        params (hi, lo)."""
        pr = np.zeros(4, dtype=np.float64)
        pr[:len(params)] = params
        flags = np.zeros(self.num_blocks, dtype=np.int32)
        ind = np.zeros(self.num_blocks, dtype=np.float64)
        self._chk(self.L.ora_refine_flags(self.h, state, criterion, var, _dp(pr), _ip(flags), _dp(ind)))
        return flags, ind

    def totals(self, state):
        out = np.zeros(self.nvar, dtype=np.float64)
        self.L.ora_totals(self.h, state, _dp(out))
        return out

    def permute(self, perm):
        p = np.ascontiguousarray(perm, dtype=np.int32)
        assert sorted(p.tolist()) == list(range(self.num_blocks))
        self.L.ora_permute(self.h, _ip(p))

    def face_table(self):
        nb, nf = self.num_blocks, 2 * self.dim
        kind = np.zeros((nb, nf), dtype=np.int32)
        nbr = np.zeros((nb, nf, 4), dtype=np.int32)
        off = np.zeros((nb, nf, 2), dtype=np.int32)
        self.L.ora_face_table(self.h, _ip(kind), _ip(nbr), _ip(off))
        return kind, nbr, off


def minmod_G(a, b, theta):
    return lib().ora_minmod_G(a, b, theta)


def vanleer(a, b):
    return lib().ora_vanleer(a, b)


def koren(a, b):
    return lib().ora_koren(a, b)


def weno3(a, b):
    return lib().ora_weno3(a, b)


def riemann_flux(dim, gamma, wL, wR, direction, flux=FLUX_HLL):
    wL = np.asarray(wL, dtype=np.float64)
    wR = np.asarray(wR, dtype=np.float64)
    F = np.zeros(dim + 2)
    lib().ora_riemann_flux(dim, gamma, flux, _dp(wL), _dp(wR), direction, _dp(F))
    return F


def wavespeeds(dim, gamma, wL, wR, direction):
    wL = np.asarray(wL, dtype=np.float64)
    wR = np.asarray(wR, dtype=np.float64)
    a, b = C.c_double(), C.c_double()
    lib().ora_wavespeeds(dim, gamma, _dp(wL), _dp(wR), direction, C.byref(a), C.byref(b))
    return a.value, b.value


def to_primitive(dim, gamma, U):
    U = np.asarray(U, dtype=np.float64)
    w = np.zeros(dim + 2)
    lib().ora_to_primitive(dim, gamma, _dp(U), _dp(w))
    return w


def to_conservative(dim, gamma, w):
    w = np.asarray(w, dtype=np.float64)
    U = np.zeros(dim + 2)
    lib().ora_to_conservative(dim, gamma, _dp(w), _dp(U))
    return U


def advection_flux(dim, vel, rhoL, rhoR, direction, flux=FLUX_HLL):
    v = np.zeros(3)
    v[:dim] = vel
    return lib().ora_advection_flux(dim, _dp(v), flux, rhoL, rhoR, direction)

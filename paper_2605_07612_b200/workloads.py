"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is the ONLY code that serves both the oracle (``oracle/``) and the
CUDA library (``paper_2605_07612_b200/csrc``).  It holds no part of the method
(no ghost rule, limiter, flux, update or reduction): it only places numbers in
cells.  The inputs stand in for the paper's Rayleigh-Taylor / advection
workloads: same shapes (uniform 256^3-768^3 in
8^3/16^3/32^3 blocks, 2 ghost layers, fp64, plus a 16^3-block AMR case); the
paper uses no public dataset.

Geometry convention (DESIGN.md "Readings" A13): the domain is
``[0, brick[a]/max(brick)]`` along axis ``a``; a block at level ``l`` with
integer block coordinates ``c`` has cubic cells of size
``dx_l = 1/(max(brick) * 2**l * N)`` and cell centres
``x = (c*N + i + 1/2) * dx_l`` for the 0-based interior index ``i``.

Noise is counter-based and order-independent (so that oracle and library may
number their blocks differently):
``u01(seed, stream, gid) = (mix64(mix64(seed ^ stream*K1) + gid*K2) >> 11) * 2**-53``
with ``mix64`` the splitmix64 finaliser and ``gid`` the linear index of the
cell on its own level's global grid (the level is folded into ``stream``).
"""
from __future__ import annotations

import numpy as np

_K1 = np.uint64(0xD6E8FEB86659FD93)
_K2 = np.uint64(0x9E3779B97F4A7C15)

PERIODIC, OUTFLOW, KEEP, DIRICHLET, NEUMANN, BCDATA = 0, 1, 2, 3, 4, 5  # values of bc_kind, same numbering as include/f4.h


def mix64(x: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on uint64 arrays (wrap-around arithmetic)."""
    x = np.asarray(x, dtype=np.uint64).copy()
    with np.errstate(over="ignore"):
        x ^= x >> np.uint64(30)
        x *= np.uint64(0xBF58476D1CE4E5B9)
        x ^= x >> np.uint64(27)
        x *= np.uint64(0x94D049BB133111EB)
        x ^= x >> np.uint64(31)
    return x


def u01(seed: int, stream: int, gid: np.ndarray) -> np.ndarray:
    """Uniform [0,1) doubles from (seed, stream, counter)."""
    gid = np.asarray(gid, dtype=np.uint64)
    with np.errstate(over="ignore"):
        s = np.uint64(seed) ^ (np.uint64(stream) * _K1)
        h = mix64(mix64(np.array([s], dtype=np.uint64))[0] + gid * _K2)
    return (h >> np.uint64(11)).astype(np.float64) * 2.0 ** -53


def sym(seed: int, stream: int, gid: np.ndarray) -> np.ndarray:
    """Uniform [-1,1)."""
    return 2.0 * u01(seed, stream, gid) - 1.0


# --------------------------------------------------------------------------
# configs
# --------------------------------------------------------------------------
def config(n: int, scale: int | None = None) -> dict:
    """Mesh + run parameters of BASELINE.json config ``n`` (1-based).

    ``scale`` (optional) replaces the uniform base level (configs 2-4) or the
    number of extra levels (config 5) to get a small case with the same
    generator for parity tests.
    """
    per = [PERIODIC] * 6
    out = [OUTFLOW] * 6
    if n == 1:
        c = dict(dim=2, block_n=8, brick=(2, 2, 1), base_level=1, max_level=1, bc=per,
                 steps=10, seed=1001, ic="sinewave")
    elif n == 2:
        c = dict(dim=3, block_n=8, brick=(1, 1, 1), base_level=5, max_level=5, bc=per,
                 steps=20, seed=1002, ic="kh")
    elif n == 3:
        c = dict(dim=3, block_n=16, brick=(1, 1, 1), base_level=5, max_level=5, bc=per,
                 steps=20, seed=1003, ic="kh")
    elif n == 4:
        c = dict(dim=3, block_n=32, brick=(3, 3, 3), base_level=3, max_level=3, bc=per,
                 steps=10, seed=1004, ic="fourier")
    elif n == 5:
        c = dict(dim=3, block_n=16, brick=(1, 1, 1), base_level=3, max_level=6, bc=out,
                 steps=100, seed=1005, ic="blast", regrid_every=10)
    elif n == 6:
        # Not a BASELINE.json config: the paper's own Euler benchmark, the Rayleigh-Taylor set-up of PAPER.md:425-431
        # as run for Table 1 (3D 512^3, 16^3 blocks, van Leer, Heun, CFL 0.5, gamma = 5/3,
        # g = (0,0,-1), periodic in x and y).  The paper does not state the top / bottom boundary condition nor the
        # pressure at the top; reading B5: uniform Neumann faces that continue the hydrostatic state of
        # a gas at rest -- d(rho)/dn = d(momentum)/dn = 0, dE/dn = -+rho g/(gamma-1) -- and p_top = 1.
        g1 = 5.0 / 3.0 - 1.0
        bcv = [[0.0] * 5 for _ in range(6)]
        bcv[4][4] = 0.1 / g1       # -z face: outward normal is -z, dE/dz = -rho_low/(gamma-1)
        bcv[5][4] = -1.0 / g1      # +z face: dE/dz = -rho_high/(gamma-1)
        c = dict(dim=3, block_n=16, brick=(1, 1, 1), base_level=5, max_level=5,
                 bc=[PERIODIC] * 4 + [NEUMANN] * 2, steps=20, seed=1006, ic="rt",
                 gravity=(0.0, 0.0, -1.0), bc_values=bcv)
    elif n == 7:
        # Not a BASELINE.json config: the paper's AMR run of the same Rayleigh-Taylor set-up (section
        # 5.4): refinement criterion eq. (12) on the gas density with c_refine = 5e-2, c_derefine = 6.25e-3,
        # eps = 1e-2, eps_abs = 1e-10, regrid every four time steps, 16^3 blocks.  Here: base level 2 (64^3 cells),
        # up to 3 more levels (the paper: levels 0-6 on 64 GPUs).
        c = config(6)
        c.update(base_level=2, max_level=5, steps=40, seed=1007, regrid_every=4,
                 criterion=("lohner", 0, (5e-2, 6.25e-3, 1e-2, 1e-10)))
        if scale is not None:
            c["max_level"] = c["base_level"] + scale
        c["name"] = "rayleigh-taylor-amr"
        return c
    elif n == 8:
        # Not a BASELINE.json config: the paper's second physics, scalar advection eq. (13) with v = (1,1,1) on the
        # periodic unit cube, initial condition eq. (17), van Leer, Heun, CFL 0.5,
        # 3D 512^3 in 16^3 blocks as in Table 1 (10.89 GCUPS on one H100)
        c = dict(dim=3, block_n=16, brick=(1, 1, 1), base_level=5, max_level=5, bc=per, steps=20, seed=1008,
                 ic="bump", physics="advection", velocity=(1.0, 1.0, 1.0))
        c.update(n_ghost=2, gamma=1.4, cfl=0.5, name="advection")
        if scale is not None:
            c["base_level"] = c["max_level"] = scale
        return c
    else:
        raise ValueError("config 1..8")
    c.update(n_ghost=2, gamma=1.4, cfl=0.4, name=f"config{n}")
    if n == 6:
        c.update(gamma=5.0 / 3.0, cfl=0.5, name="rayleigh-taylor")
        if scale is not None:
            c["base_level"] = c["max_level"] = scale
        return c
    if scale is not None:
        if n == 5:
            c["max_level"] = c["base_level"] + scale
        else:
            c["base_level"] = c["max_level"] = scale
    return c


# --------------------------------------------------------------------------
# geometry helpers
# --------------------------------------------------------------------------
def cell_centres(cfg: dict, levels: np.ndarray, coords: np.ndarray):
    """Cell-centre coordinates and global cell ids of every interior cell.

    levels: [nb] int, coords: [nb,3] int (block coordinates on the level's grid).
    Returns (xyz, gid): xyz is a list of dim arrays shaped [nb, Nz, Ny, Nx]
    (Nz=1 in 2D), gid a uint64 array of the same shape.
    """
    dim, n = cfg["dim"], cfg["block_n"]
    levels = np.asarray(levels, dtype=np.int64)
    coords = np.asarray(coords, dtype=np.int64).reshape(-1, 3)
    nb = levels.shape[0]
    maxb = max(cfg["brick"][:dim])
    dx = 1.0 / (maxb * (2.0 ** levels) * n)  # [nb]
    nz = n if dim == 3 else 1
    shape = (nb, nz, n, n)
    ar = np.arange(n, dtype=np.int64)
    gi = (coords[:, 0, None] * n + ar[None, :])[:, None, None, :]
    gj = (coords[:, 1, None] * n + ar[None, :])[:, None, :, None]
    if dim == 3:
        gk = (coords[:, 2, None] * n + ar[None, :])[:, :, None, None]
    else:
        gk = np.zeros((nb, 1, 1, 1), dtype=np.int64)
    d = dx[:, None, None, None]
    xyz = [np.broadcast_to((gi + 0.5) * d, shape), np.broadcast_to((gj + 0.5) * d, shape)]
    if dim == 3:
        xyz.append(np.broadcast_to((gk + 0.5) * d, shape))
    ext = [cfg["brick"][a] * n * (2 ** levels) for a in range(3)]  # cells per axis on level
    ex = ext[0][:, None, None, None]
    ey = ext[1][:, None, None, None]
    gid = ((gk * ey + gj) * ex + gi).astype(np.uint64)
    return xyz, np.broadcast_to(gid, shape)


def _level_stream(base: int, levels: np.ndarray, shape) -> np.ndarray:
    return np.broadcast_to((base * 64 + np.asarray(levels, dtype=np.int64))[:, None, None, None], shape)


def _noise(seed: int, base_stream: int, levels, gid) -> np.ndarray:
    """sym() with the level folded into the stream id (one stream per level)."""
    out = np.empty(gid.shape, dtype=np.float64)
    levels = np.asarray(levels)
    for l in np.unique(levels):
        m = levels == l
        out[m] = sym(seed, base_stream * 64 + int(l), gid[m])
    return out


# --------------------------------------------------------------------------
# initial states (primitive variables rho, u[dim], p), shape [nb, nvar, Nz, Ny, Nx]
# --------------------------------------------------------------------------
def blast_centre(cfg: dict) -> np.ndarray:
    s = sym(cfg["seed"], 7, np.arange(3, dtype=np.uint64))
    return 0.5 + s / 128.0


def fourier_modes(cfg: dict):
    """8 seeded modes: integer wave vectors in {1..4}^3 and phases in [0,2pi)."""
    seed = cfg["seed"]
    k = 1 + np.floor(4.0 * u01(seed, 11, np.arange(24, dtype=np.uint64))).astype(np.int64).reshape(8, 3)
    phi = 2.0 * np.pi * u01(seed, 12, np.arange(8, dtype=np.uint64))
    return k, phi


def initial_primitives(cfg: dict, levels, coords, noise: bool = True) -> np.ndarray:
    dim = cfg["dim"]
    nvar = dim + 2
    xyz, gid = cell_centres(cfg, levels, coords)
    shape = gid.shape
    w = np.zeros((shape[0], nvar) + shape[1:], dtype=np.float64)
    seed = cfg["seed"]
    ic = cfg["ic"]
    x, y = xyz[0], xyz[1]
    if ic == "sinewave":  # config 1
        w[:, 0] = 1.0 + 0.1 * np.sin(2 * np.pi * x) * np.sin(2 * np.pi * y)
        if noise:
            w[:, 0] += 1e-3 * _noise(seed, 1, levels, gid)
        w[:, 1] = 0.5
        w[:, 2] = 0.5
        w[:, nvar - 1] = 1.0
    elif ic == "kh":  # configs 2, 3
        inner = np.abs(y - 0.5) < 0.25
        w[:, 0] = np.where(inner, 2.0, 1.0)
        w[:, 1] = np.where(inner, 0.5, -0.5)
        w[:, 2] = 0.01 * _noise(seed, 2, levels, gid) if noise else 0.0
        w[:, nvar - 1] = 2.5
    elif ic == "fourier":  # config 4
        z = xyz[2]
        k, phi = fourier_modes(cfg)
        rho = np.ones(shape, dtype=np.float64)
        for m in range(8):
            rho += (0.05 / 8.0) * np.sin(2 * np.pi * (k[m, 0] * x + k[m, 1] * y + k[m, 2] * z) + phi[m])
        w[:, 0] = rho
        for a in range(3):
            w[:, 1 + a] = 0.1 * _noise(seed, 3 + a, levels, gid) if noise else 0.0
        w[:, nvar - 1] = 1.0
    elif ic == "blast":  # config 5
        z = xyz[2]
        c = blast_centre(cfg)
        r2 = (x - c[0]) ** 2 + (y - c[1]) ** 2 + (z - c[2]) ** 2
        w[:, 0] = 1.0
        w[:, nvar - 1] = np.where(r2 < 0.05 ** 2, 100.0, 1e-2)
    elif ic == "rt":  # heavy (rho = 1) over light (rho = 0.1) fluid, interface at
        # h(x,y) = 0.8 + 0.05 sin(2 pi x) sin(2 pi y), at rest, pressure in hydrostatic balance with g = (0,0,-1)
        z = xyz[2]
        h = 0.8 + 0.05 * np.sin(2 * np.pi * x) * np.sin(2 * np.pi * y)
        above = z > h
        w[:, 0] = np.where(above, 1.0, 0.1)
        w[:, nvar - 1] = np.where(above, 1.0 + 1.0 * (1.0 - z), 1.0 + 1.0 * (1.0 - h) + 0.1 * (h - z))
    elif ic == "uniform":
        w[:, 0] = cfg.get("rho0", 1.0)
        for a in range(dim):
            w[:, 1 + a] = cfg.get("vel0", (0.0, 0.0, 0.0))[a]
        w[:, nvar - 1] = cfg.get("p0", 1.0)
    else:
        raise ValueError(ic)
    return w


def prim_to_cons(w: np.ndarray, gamma: float) -> np.ndarray:
    """Input formatting: the state handed to ``set_state`` is conservative
    (rho, rho*u, E) with E from PAPER.md:380 eq. (15)."""
    nvar = w.shape[1]
    dim = nvar - 2
    u = np.empty_like(w)
    rho = w[:, 0]
    u[:, 0] = rho
    ke = np.zeros_like(rho)
    for a in range(dim):
        u[:, 1 + a] = rho * w[:, 1 + a]
        ke = ke + w[:, 1 + a] * w[:, 1 + a]
    u[:, nvar - 1] = w[:, nvar - 1] / (gamma - 1.0) + 0.5 * rho * ke
    return u


def scalar_field(cfg: dict, levels, coords) -> np.ndarray:
    """Scalar advection inputs (one variable), [nb, 1, Nz, Ny, Nx]: the paper's compact bump eq. (17) (PAPER.md:398:
    R = 0.1, delta = 0.05) or the Gaussian of its convergence test eq. (19) (R = 0.1), both centred in the
    unit domain, evaluated at the cell centres."""
    xyz, gid = cell_centres(cfg, levels, coords)
    d2 = sum((c - 0.5) ** 2 for c in xyz)
    if cfg["ic"] == "gauss":
        rho = np.exp(-d2 / 0.1 ** 2)
    elif cfg["ic"] == "bump":
        R, delta = 0.1, 0.05
        d = np.sqrt(d2)
        q = 1.0 + (d - R) / delta
        rho = np.where(d < R - delta, 1.0, np.where(d < R, 1.0 - 3.0 * q ** 2 + 2.0 * q ** 3, 0.0))
    else:
        raise ValueError(cfg["ic"])
    return np.ascontiguousarray(np.broadcast_to(rho, gid.shape)[:, None].astype(np.float64))


def initial_state(cfg: dict, levels, coords, noise: bool = True) -> np.ndarray:
    """Conservative interior state [nb, nvar, Nz, Ny, Nx] (C-contiguous)."""
    if cfg.get("physics") == "advection":
        return scalar_field(cfg, levels, coords)
    return np.ascontiguousarray(prim_to_cons(initial_primitives(cfg, levels, coords, noise), cfg["gamma"]))


def apply_physics(cfg: dict, mesh) -> None:
    """Hand the config's run-time options (gravity, uniform boundary values) to a mesh object of either
    implementation (same method names); argument passing only."""
    if "gravity" in cfg:
        mesh.set_gravity(cfg["gravity"])
    if "bc_values" in cfg:
        nvar = cfg["dim"] + 2
        mesh.set_bc_values(np.asarray(cfg["bc_values"], dtype=np.float64)[:, :nvar])


def uniform_blocks(cfg: dict):
    """(levels, coords) of the uniform base-level mesh in x-fastest raster order.
    Only used to size host buffers; both implementations report their own order."""
    l = cfg["base_level"]
    ext = [cfg["brick"][a] * 2 ** l for a in range(3)]
    if cfg["dim"] == 2:
        ext[2] = 1
    kk, jj, ii = np.meshgrid(np.arange(ext[2]), np.arange(ext[1]), np.arange(ext[0]), indexing="ij")
    coords = np.stack([ii.ravel(), jj.ravel(), kk.ravel()], axis=1).astype(np.int32)
    return np.full(coords.shape[0], l, dtype=np.int32), coords

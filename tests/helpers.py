"""Test-side helpers: geometry of padded blocks, brute-force mesh checks,
block matching between two implementations.  No method arithmetic."""
from __future__ import annotations

import itertools

import numpy as np


def padded_coords(dim, N, Ng, brick, levels, coords):
    """Cell-centre coordinates of every padded cell, natural layout
    [nb, Pz, Py, Px] per axis, plus masks:
      noncorner: at most one index outside the interior (cells the method uses)
      outside:   cell centre lies outside the domain (physical-boundary ghost)"""
    P = N + 2 * Ng
    nb = len(levels)
    maxb = max(brick[:dim])
    dx = 1.0 / (maxb * 2.0 ** np.asarray(levels, dtype=np.float64) * N)
    idx = np.arange(-Ng, N + Ng)
    Pz = P if dim == 3 else 1
    shape = (nb, Pz, P, P)
    X = np.empty((dim,) + shape)
    out_of = np.zeros(shape, dtype=np.int32)
    outside = np.zeros(shape, dtype=bool)
    for a in range(dim):
        g = (np.asarray(coords)[:, a, None] * N + idx[None, :] + 0.5) * dx[:, None]  # [nb, P]
        length = brick[a] / maxb
        sh = [nb, 1, 1, 1]
        sh[3 - a] = P
        X[a] = np.broadcast_to(g.reshape(sh), shape)
        oo = ((idx < 0) | (idx >= N)).astype(np.int32)
        sh2 = [1, 1, 1, 1]
        sh2[3 - a] = P
        out_of = out_of + oo.reshape(sh2)
        outside |= (X[a] < 0.0) | (X[a] > length)
    return X, out_of <= 1, outside


def key_index(levels, coords):
    return {(int(l), int(c[0]), int(c[1]), int(c[2])): b for b, (l, c) in enumerate(zip(levels, coords))}


def match_blocks(lev_a, co_a, lev_b, co_b):
    """perm such that block q of A is block perm[q] of B (same key)."""
    ib = key_index(lev_b, co_b)
    assert len(ib) == len(lev_b)
    return np.array([ib[(int(l), int(c[0]), int(c[1]), int(c[2]))] for l, c in zip(lev_a, co_a)], dtype=np.int64)


def check_mesh_valid(dim, brick, bc, levels, coords, base_level, max_level):
    """Brute force: leaves tile the domain exactly and every pair of leaves that
    touch (face, edge or corner, with periodic images) differs by <= 1 level."""
    levels = np.asarray(levels)
    coords = np.asarray(coords)
    assert levels.min() >= base_level and levels.max() <= max_level
    L = int(levels.max())
    ext = [brick[a] << L for a in range(dim)]
    lo = np.stack([coords[:, a] << (L - levels) for a in range(dim)], axis=1)
    size = (1 << (L - levels))
    vol = float(np.sum(size.astype(np.float64) ** dim))
    assert vol == float(np.prod(ext)), "leaves do not tile the domain volume"
    # no overlaps: paint (only for small meshes)
    if np.prod(ext) <= 2 ** 21:
        grid = np.zeros(ext[::-1], dtype=np.int32)
        for b in range(len(levels)):
            sl = tuple(slice(lo[b, a], lo[b, a] + size[b]) for a in reversed(range(dim)))
            grid[sl] += 1
        assert grid.min() == 1 and grid.max() == 1, "overlap or hole"
    # 2:1 over closed-box contact with periodic images
    shifts = []
    for a in range(dim):
        shifts.append([-ext[a], 0, ext[a]] if bc[2 * a] == 0 else [0])
    hi = lo + size[:, None]
    nb = len(levels)
    for sh in itertools.product(*shifts):
        lo_s = lo + np.asarray(sh)[None, :]
        hi_s = hi + np.asarray(sh)[None, :]
        touch = np.ones((nb, nb), dtype=bool)
        for a in range(dim):
            touch &= (lo[:, None, a] <= hi_s[None, :, a]) & (lo_s[None, :, a] <= hi[:, None, a])
        dl = np.abs(levels[:, None] - levels[None, :])
        bad = touch & (dl > 1)
        assert not bad.any(), f"2:1 balance violated for pairs {np.argwhere(bad)[:4]}"


def rel_linf(a, b):
    """Reading A16: per variable max|a-b| / max|b| over all interior cells."""
    nvar = a.shape[1]
    out = np.zeros(nvar)
    for v in range(nvar):
        den = np.abs(b[:, v]).max()
        num = np.abs(a[:, v] - b[:, v]).max()
        out[v] = num / den if den > 0 else num
    return out


# --------------------------------------------------------------------------
# config-5 refinement rule, reading A15, as a vectorised numpy statement: cross-check of the oracle's cell loop
# --------------------------------------------------------------------------
def pressure_jump_flags_numpy(cfg: dict, padded: np.ndarray, hi: float = 0.1, lo: float = 0.025) -> np.ndarray:
    """Flags from a ghost-filled conservative state in natural padded layout
    [nb, nvar, Pz, Py, Px].  J = max over face-adjacent cell pairs
    (interior-interior and interior-first ghost layer) of |pa-pb|/min(pa,pb);
    +1 if J>hi, -1 if J<lo, else 0."""
    dim, n, ng, gamma = cfg["dim"], cfg["block_n"], cfg["n_ghost"], cfg["gamma"]
    nvar = dim + 2
    rho = padded[:, 0]
    ke = np.zeros_like(rho)
    with np.errstate(all="ignore"):
        for a in range(dim):
            ke = ke + padded[:, 1 + a] ** 2
        p = (gamma - 1.0) * (padded[:, nvar - 1] - 0.5 * ke / rho)
    nb = padded.shape[0]
    J = np.zeros(nb)
    lo_i, hi_i = ng, ng + n  # interior slice
    ints = [slice(lo_i, hi_i)] * 3
    if dim == 2:
        ints[0] = slice(0, 1)
    for a in range(dim):
        ax = 3 - a  # array axis in [nb, z, y, x]
        sl_a = [slice(None)] + list(ints)
        sl_b = [slice(None)] + list(ints)
        sl_a[ax] = slice(lo_i - 1, hi_i)      # cells -1 .. N-1
        sl_b[ax] = slice(lo_i, hi_i + 1)      # cells  0 .. N
        pa, pb = p[tuple(sl_a)], p[tuple(sl_b)]
        with np.errstate(all="ignore"):
            jump = np.abs(pa - pb) / np.minimum(pa, pb)
        J = np.maximum(J, jump.reshape(nb, -1).max(axis=1))
    flags = np.zeros(nb, dtype=np.int32)
    flags[J > hi] = 1
    flags[J < lo] = -1
    return flags


def boundary_faces(dim, N, brick, bc, levels, coords, kind):
    """(block, face) pairs on the physical boundary whose face direction has bc kind `kind`, in (block, face) order,
    and the cell-centre coordinates of their face cells: xyz[q][axis] arrays shaped [kmax, N] (t2, t1), with the
    coordinate along the face normal set ON the face."""
    maxb = max(brick[:dim])
    out, xyz = [], []
    for b, (l, c) in enumerate(zip(levels, coords)):
        dx = 1.0 / (maxb * 2.0 ** int(l) * N)
        for f in range(2 * dim):
            a, side = f // 2, f % 2
            ext = brick[a] * 2 ** int(l)
            if bc[f] != kind or (c[a] != (ext - 1 if side else 0)):
                continue
            ta = [ax for ax in range(dim) if ax != a]
            kmax = N if dim == 3 else 1
            t1 = (c[ta[0]] * N + np.arange(N) + 0.5) * dx
            X = [None] * 3
            X[a] = np.full((kmax, N), (c[a] + side) * N * dx)
            X[ta[0]] = np.broadcast_to(t1[None, :], (kmax, N)).copy()
            if dim == 3:
                t2 = (c[ta[1]] * N + np.arange(N) + 0.5) * dx
                X[ta[1]] = np.broadcast_to(t2[:, None], (kmax, N)).copy()
            else:
                X[2] = np.zeros((kmax, N))
            out.append((b, f))
            xyz.append(X)
    return out, xyz

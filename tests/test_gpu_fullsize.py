"""GPU parity at BASELINE.json's FULL sizes (-m gpu), in the launch configuration bench.py times
(f4.Mesh.from_config -> bind_torch -> set_state -> compute_dt/advance).

The oracle cannot run 512^3 cells in seconds, so the full-size runs are checked
 (a) on SAMPLED blocks the oracle computes one by one: one Heun step of a block depends only on the
     cells within 2 x 2 = 4 cells of it, i.e. on its 26 neighbours' interiors.  The 3^3 (or 4^3)
     patch of blocks around a sampled block is copied out of the GPU state BEFORE the step into a
     small periodic oracle mesh, advanced by the oracle with the same dt/dx, and its centre block is
     compared element by element with the GPU state AFTER the step (1e-11 relative L-inf, reading A16);
 (b) via properties that hold at any size: conserved totals of the periodic run constant to 1e-12
     relative, positivity, and compute_dt against the definition evaluated with numpy on the state.
"""
from __future__ import annotations

import numpy as np
import pytest

import helpers as H
from oracle import oracle as O
from paper_2605_07612_b200 import f4
from paper_2605_07612_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL_STATE, TOL_TOTALS = 1e-11, 1e-12


def _fill(cfg, lev, co, out, chunk=2048):
    for b0 in range(0, len(lev), chunk):
        out[b0:b0 + chunk] = W.initial_state(cfg, lev[b0:b0 + chunk], co[b0:b0 + chunk])


def _rate_by_definition(u, gamma, dx):
    """max over cells of sum_d (|u_d| + c)/dx (reading A5), chunked numpy on the interior state."""
    best = 0.0
    nvar = u.shape[1]
    for b0 in range(0, u.shape[0], 1024):
        s = u[b0:b0 + 1024]
        rho = s[:, 0]
        ke = sum(s[:, 1 + a] ** 2 for a in range(nvar - 2))
        p = (gamma - 1.0) * (s[:, nvar - 1] - 0.5 * ke / rho)
        c = np.sqrt(gamma * p / rho)
        r = sum(np.abs(s[:, 1 + a]) / rho + c for a in range(nvar - 2)) / dx
        best = max(best, float(r.max()))
    return best


@pytest.mark.parametrize("n,warm_steps,nsample", [(2, 2, 6), (3, 2, 6), (4, 1, 4)])
def test_full_size_sampled_blocks_and_invariants(n, warm_steps, nsample):
    cfg = W.config(n)
    N, dim, gamma = cfg["block_n"], cfg["dim"], cfg["gamma"]
    lm = f4.Mesh.from_config(cfg)
    lm.bind_torch()
    lev, co = lm.get_blocks()
    nb = len(lev)
    ext = [cfg["brick"][a] << cfg["base_level"] for a in range(3)]
    assert nb == ext[0] * ext[1] * ext[2]
    u = np.empty(lm._shape(False))
    _fill(cfg, lev, co, u)
    lm.set_state(0, u)
    t0 = lm.conserved_totals(0)
    for _ in range(warm_steps):
        lm.advance(lm.compute_dt(0, cfg["cfl"]))
    before = lm.get_state(0, out=u)
    dx = 1.0 / (max(cfg["brick"]) * 2 ** cfg["base_level"] * N)
    dt = lm.compute_dt(0, cfg["cfl"])
    # (b) compute_dt against the definition on the same state
    rate = _rate_by_definition(before, gamma, dx)
    assert abs(dt - cfg["cfl"] / rate) <= 1e-13 * dt
    lm.advance(dt)
    after = lm.get_state(0)
    t1 = lm.conserved_totals(0)
    scale = np.abs(t0).max()
    assert np.all(np.abs(t1 - t0) <= TOL_TOTALS * scale), (t1 - t0) / scale
    assert after[:, 0].min() > 0.0
    den = np.array([np.abs(after[:, v]).max() for v in range(dim + 2)])

    # (a) sampled blocks: the patch side m divides the block-grid extent into a power of two, so dt/dx is kept exactly
    m = 3 if (ext[0] % 3 == 0) else 4
    ratio = ext[0] / m
    assert ratio == 2.0 ** round(np.log2(ratio)) and len(set(ext)) == 1
    pcfg = dict(dim=3, block_n=N, n_ghost=2, brick=(m, m, m), base_level=0, max_level=0, bc=[W.PERIODIC] * 6,
                gamma=gamma)
    index = H.key_index(lev, co)
    rng = np.random.default_rng(4200 + n)
    picks = [0, nb - 1] + [int(x) for x in rng.integers(0, nb, nsample - 2)]
    worst = np.zeros(dim + 2)
    for b in picks:
        om = O.OracleMesh.from_config(pcfg)
        lo, cob = om.get_blocks()
        patch = np.empty((len(lo),) + before.shape[1:])
        centre = None
        for q, c in enumerate(cob):
            src = tuple((int(co[b][a]) + int(c[a]) - 1) % ext[a] for a in range(3))
            patch[q] = before[index[(int(lev[b]),) + src]]
            if tuple(int(x) for x in c) == (1, 1, 1):
                centre = q
        om.set_state(0, patch)
        om.advance(dt * ratio)          # same dt/dx: the patch's cells are `ratio` times larger
        ref = om.get_state(0)[centre]
        err = np.array([np.abs(after[b, v] - ref[v]).max() for v in range(dim + 2)]) / den
        worst = np.maximum(worst, err)
        assert np.all(err <= TOL_STATE), (b, err)
    print(f"config{n}: {len(picks)} sampled blocks, worst rel L-inf per variable {worst}")
    lm.close()

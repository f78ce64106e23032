"""GPU parity of the scalar advection path (-m gpu; eq. (13), tests of PAPER.md:396-421): the CUDA
kernels through the C-ABI against the oracle on the same inputs; state <= 1e-11 (A16), totals <= 1e-12."""
from __future__ import annotations

import numpy as np
import pytest

import helpers as H
from oracle import oracle as O
from paper_2605_07612_b200 import f4
from paper_2605_07612_b200 import workloads as W

pytestmark = pytest.mark.gpu
PER, OUT = W.PERIODIC, W.OUTFLOW
TOL_STATE, TOL_TOTALS = 1e-11, 1e-12


def adv_cfg(dim, N, brick, level, max_level=None, ic="bump", vel=None, bc=None):
    return dict(dim=dim, block_n=N, n_ghost=2, brick=tuple(brick) + (1,) * (3 - len(brick)), base_level=level,
                max_level=level if max_level is None else max_level, bc=bc or [PER] * (2 * dim), gamma=1.4, cfl=0.5,
                ic=ic, physics="advection", velocity=vel or (1.0,) * dim, seed=1, name="adv")


def pair(cfg, max_blocks=None):
    lm = f4.Mesh.from_config(cfg, max_blocks=max_blocks)
    lm.bind_torch()
    om = O.OracleMesh.from_config(cfg)
    assert lm.nvar == 1 and om.nvar == 1
    return lm, om


def perm_of(lm, om):
    la, ca = lm.get_blocks()
    lb, cb = om.get_blocks()
    return H.match_blocks(la, ca, lb, cb)


def set_both(lm, om, cfg, u=None):
    la, ca = lm.get_blocks()
    if u is None:
        u = W.initial_state(cfg, la, ca)
    perm = perm_of(lm, om)
    uo = np.empty_like(u)
    uo[perm] = u
    lm.set_state(0, u)
    om.set_state(0, uo)
    return perm


def run(lm, om, cfg, perm, steps, scheme=None):
    t0 = om.totals(0)
    for _ in range(steps):
        dt = om.compute_dt(0, cfg["cfl"])
        assert abs(lm.compute_dt(0, cfg["cfl"]) - dt) <= 1e-15 * dt
        om.advance(dt, scheme)
        lm.advance(dt)
    ug, uo = lm.get_state(0), om.get_state(0)[perm]
    err = H.rel_linf(ug, uo)
    assert np.all(err <= TOL_STATE), err
    tg, to = lm.conserved_totals(0), om.totals(0)
    assert np.all(np.abs(tg - to) <= TOL_TOTALS * max(np.abs(to).max(), 1e-300))
    return t0, tg


@pytest.mark.parametrize("dim,N,brick,level,vel", [
    (2, 8, (2, 2), 1, (1.0, 1.0)), (2, 16, (3, 2), 0, (1.0, -0.5)), (2, 32, (1, 1), 1, (-1.0, 1.0)),
    (3, 8, (3, 1, 2), 1, (1.0, 1.0, 1.0)), (3, 16, (1, 1, 1), 1, (1.0, -1.0, 0.5)), (3, 16, (1, 2, 1), 0, (-1.0, 0.0, 1.0)),
    (3, 32, (1, 1, 1), 1, (1.0, 1.0, -1.0)), (3, 8, (1, 1, 1), 0, (0.3, 0.7, -1.0))])
def test_uniform_mesh_parity_and_conservation(dim, N, brick, level, vel):
    cfg = adv_cfg(dim, N, brick, level, vel=vel)
    lm, om = pair(cfg)
    rng = np.random.default_rng(N + dim)
    la, ca = lm.get_blocks()
    u = W.initial_state(cfg, la, ca) + 0.05 * rng.uniform(size=lm._shape(False))   # bump + noise: every limiter branch
    perm = set_both(lm, om, cfg, u)
    t0, tg = run(lm, om, cfg, perm, 10)
    assert abs(tg[0] - t0[0]) <= TOL_TOTALS * abs(t0[0])      # periodic: conserved
    lm.close()


@pytest.mark.parametrize("limiter", [f4.LIM_MINMOD, f4.LIM_MC])
@pytest.mark.parametrize("dim,N", [(2, 16), (3, 8)])
def test_limiter_variants(dim, N, limiter):
    cfg = adv_cfg(dim, N, (2, 2, 2)[:dim], 0)
    lm, om = pair(cfg)
    lm.set_options(limiter=limiter)
    om.set_options(limiter=limiter)
    rng = np.random.default_rng(3)
    u = rng.uniform(0.0, 1.0, lm._shape(False))
    perm = set_both(lm, om, cfg, u)
    run(lm, om, cfg, perm, 5)
    lm.close()


@pytest.mark.parametrize("scheme", [f4.RK_EULER, f4.RK_SSP33, f4.RK_SSP43])
def test_rk_schemes(scheme):
    cfg = adv_cfg(3, 8, (2, 2, 2), 0)
    lm = f4.Mesh.from_config(cfg, n_states=f4.RK_STATES[scheme])
    lm.bind_torch()
    lm.set_rk_scheme(scheme)
    om = O.OracleMesh.from_config(cfg, n_states=f4.RK_STATES[scheme])
    perm = set_both(lm, om, cfg)
    run(lm, om, cfg, perm, 4, scheme)
    lm.close()


@pytest.mark.parametrize("dim,N,bc", [(2, 8, [PER] * 4), (2, 16, [OUT] * 4), (3, 8, [PER] * 6),
                                       (3, 16, [OUT, OUT, PER, PER, OUT, OUT])])
@pytest.mark.parametrize("flux_fix", [False, True])
def test_amr_parity_ghosts_and_flux_fixing(dim, N, bc, flux_fix):
    """Refined mesh: ghost fill (SRL / BC / F2C bit-exact, C2F to 4 ulp), 8 steps with and without flux fixing
    (the paper's test of it is this scalar problem)."""
    cfg = adv_cfg(dim, N, (2, 2, 2)[:dim], 0, max_level=2, bc=bc)
    lm, om = pair(cfg, max_blocks=600)
    rng = np.random.default_rng(7)
    for _ in range(2):
        la, _ = lm.get_blocks()
        flags = (rng.uniform(size=len(la)) < 0.3).astype(np.int32)
        flags[0] = 1
        perm = perm_of(lm, om)
        fo = np.empty_like(flags)
        fo[perm] = flags
        assert lm.adapt(flags) == om.adapt(fo)
    la, ca = lm.get_blocks()
    u = W.initial_state(cfg, la, ca) + 0.05 * rng.uniform(size=lm._shape(False))
    perm = set_both(lm, om, cfg, u)
    lm.fill_ghosts(0)
    om.fill_ghosts(0)
    pg, po = lm.get_state(0, with_ghosts=True), om.get_state(0, with_ghosts=True)[perm]
    _, nc, _ = H.padded_coords(dim, N, 2, (2, 2, 2)[:dim] + (1,) * (3 - dim), la, ca)
    assert np.abs(pg[:, 0] - po[:, 0])[nc].max() <= 4 * np.spacing(2.0)
    lm.set_flux_fix(flux_fix)
    om.set_flux_fix(flux_fix)
    t0, tg = run(lm, om, cfg, perm, 8)
    if flux_fix and all(b == PER for b in bc):
        assert abs(tg[0] - t0[0]) <= 1e-13 * abs(t0[0])     # e_cons eq. (18) at round-off with the fix
    lm.close()


def test_regrid_with_lohner_flags_bit_exact():
    # eq. (12) on the advected scalar decides the mesh: flags and indicators bit-exact, transfer bit-exact for copies
    cfg = adv_cfg(3, 8, (2, 2, 2), 0, max_level=2)
    lm, om = pair(cfg, max_blocks=800)
    params = (5e-2, 6.25e-3, 1e-2, 1e-10)
    for _ in range(2):
        perm = set_both(lm, om, cfg)
        om.fill_ghosts(0)
        fo, io = om.refine_flags(0, om.CRIT_LOHNER, params, 0)
        fg, ig = lm.refine_flags(0, f4.CRIT_LOHNER, params, 0)
        assert np.array_equal(fg, fo[perm]) and np.array_equal(ig, io[perm])
        assert lm.adapt(fg) == om.adapt(fo)
    perm = set_both(lm, om, cfg)
    assert lm.get_blocks()[0].max() == 2
    run(lm, om, cfg, perm, 6)
    lm.close()

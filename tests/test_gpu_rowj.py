"""GPU parity at the sizes BASELINE.json states (-m gpu): config 5 on its own mesh (base 8^3 blocks of 16^3,
three extra levels) against the oracle, and the paper's linear-field test through the CUDA
path on reference points of every class (corner, edge, face, centre), three levels deep, 32^d blocks included."""
from __future__ import annotations

import itertools

import numpy as np
import pytest

import helpers as H
from oracle import oracle as O
from paper_2605_07612_b200 import f4
from paper_2605_07612_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL_STATE, TOL_TOTALS = 1e-11, 1e-12
PJUMP = (0.1, 0.025)


def _perm(lm, om):
    la, ca = lm.get_blocks()
    lb, cb = om.get_blocks()
    return H.match_blocks(la, ca, lb, cb)


def _set_both(lm, om, cfg):
    la, ca = lm.get_blocks()
    u = W.initial_state(cfg, la, ca)
    lm.set_state(0, u)
    perm = _perm(lm, om)
    uo = np.empty_like(u)
    uo[perm] = u
    om.set_state(0, uo)
    return perm


@pytest.mark.timeout(1200)
def test_config5_on_its_baseline_mesh():
    """BASELINE.json config 5 as bench.py builds it (W.config(5): base level 3 = 8^3 blocks of 16^3 cells, up to
    three more levels, outflow, blast; initial mesh by {analytic state, flag, adapt} x 3, reading A15), 10 Heun
    steps at CFL 0.4 with a regrid after step 5; the refinement flags come from the oracle state and go to both
    adapts (reading A15).  State <= 1e-11 (A16), totals <= 1e-12, dt <= 1e-12 along the run."""
    cfg = W.config(5)
    lm = f4.Mesh.from_config(cfg, max_blocks=6000)
    lm.bind_torch()
    om = O.OracleMesh.from_config(cfg)
    for _ in range(cfg["max_level"] - cfg["base_level"]):
        perm = _set_both(lm, om, cfg)
        om.fill_ghosts(0)
        fo, _ = om.refine_flags(0, om.CRIT_PJUMP, PJUMP)
        ch_o, ch_g = om.adapt(fo), lm.adapt(fo[perm])
        assert ch_o == ch_g
        if not ch_o:
            break
    perm = _set_both(lm, om, cfg)
    lev = lm.get_blocks()[0]
    assert lev.min() == 3 and lev.max() == 6 and lm.num_blocks > 1500     # the bench's mesh: 1 772 blocks
    rec, n1, n2 = lm.pattern()
    assert n2 > 0 and (rec[:, 0] == f4.OP_F2C).any() and (rec[:, 0] == f4.OP_BC).any()
    nb0 = lm.num_blocks
    for s in range(10):
        if s == 5:
            om.fill_ghosts(0)
            fo, io = om.refine_flags(0, om.CRIT_PJUMP, PJUMP)
            fg, ig = lm.refine_flags(0, f4.CRIT_PJUMP, PJUMP)
            # device flags differ from the oracle's only where the indicator sits on a threshold
            near = np.minimum(np.abs(io[perm] - PJUMP[0]), np.abs(io[perm] - PJUMP[1])) <= 1e-9
            assert not np.any((fg != fo[perm]) & ~near)
            ch_o, ch_g = om.adapt(fo), lm.adapt(fo[perm])
            assert ch_o == ch_g
            perm = _perm(lm, om)
            assert np.all(H.rel_linf(lm.get_state(0), om.get_state(0)[perm]) <= TOL_STATE)
            print("regrid changed the mesh:", bool(ch_o), nb0, "->", lm.num_blocks, "blocks")
        dt = om.compute_dt(0, cfg["cfl"])
        assert abs(lm.compute_dt(0, cfg["cfl"]) - dt) <= 1e-12 * dt
        om.advance(dt)
        lm.advance(dt)
    err = H.rel_linf(lm.get_state(0), om.get_state(0)[perm])
    print("config 5 at size, 10 steps: rel Linf", err)
    assert np.all(err <= TOL_STATE), err
    tg, to = lm.conserved_totals(0), om.totals(0)
    assert np.all(np.abs(tg - to) <= TOL_TOTALS * np.abs(to).max())
    lm.close()


def _reference_points(dim):
    """The paper's reference points have coordinates in {0.01, 0.5, 0.99}: four of each class that has
    four (corner: no 0.5, edge: one 0.5, face: two 0.5 in 3D) and the centre."""
    pts = {}
    for p in itertools.product((0.01, 0.5, 0.99), repeat=dim):
        pts.setdefault(sum(c == 0.5 for c in p), []).append(p)
    out = []
    for nhalf in sorted(pts):
        group = pts[nhalf]
        # spread the picks over the group (first, last and two in between)
        idx = sorted({0, len(group) // 3, (2 * len(group)) // 3, len(group) - 1})
        out += [group[i] for i in idx]
    return out


@pytest.mark.timeout(1800)
@pytest.mark.parametrize("dim,N,levels", [(2, 8, 3), (2, 32, 3), (3, 16, 3), (3, 32, 3)])
def test_linear_field_reference_points(dim, N, levels):
    """phi = x + 2y + 3z in every variable, domain-boundary ghosts preset analytically (BC kind KEEP), refine `levels`
    times around a reference point and coarsen back; after every mesh change all face ghosts and all interior cells
    are phi to 4 ulp of max|phi| (limiter inactive: G(a,a)=a; eq. 21-22)."""
    tol = 4 * np.spacing(6.0)
    brick = (2, 2, 2)[:dim]
    pts = _reference_points(dim)
    assert len(pts) >= (9 if dim == 2 else 13)
    m = f4.Mesh(dim, N, 2, brick, 0, levels, [W.KEEP] * (2 * dim), max_blocks=700 if N < 32 or dim == 2 else 260)
    m.bind_torch()

    def lin(X):
        return X[0] + 2 * X[1] + (3 * X[2] if dim == 3 else 0.0)

    def check():
        lev, co = m.get_blocks()
        X, noncorner, outside = H.padded_coords(dim, N, 2, brick, lev, co)
        phi = lin(X)
        u = m.get_state(0, with_ghosts=True)
        for v in range(m.nvar):
            u[:, v] = np.where(outside, phi, u[:, v])
        m.set_state(0, u, with_ghosts=True)
        m.fill_ghosts(0)
        u = m.get_state(0, with_ghosts=True)
        for v in range(m.nvar):
            assert np.abs(u[:, v] - phi)[noncorner].max() <= tol

    lev, co = m.get_blocks()
    X, _, _ = H.padded_coords(dim, N, 2, brick, lev, co)
    m.set_state(0, np.repeat(lin(X)[:, None], m.nvar, axis=1), with_ghosts=True)
    check()
    for rref in pts:
        for _ in range(levels):
            lev, co = m.get_blocks()
            size = 1.0 / (2 * 2.0 ** lev)
            flags = np.ones(len(lev), dtype=np.int32)
            for a in range(dim):
                lo = co[:, a] * size
                flags &= ((lo <= rref[a]) & (rref[a] < lo + size)).astype(np.int32)
            assert m.adapt(flags)
            check()
        assert m.get_blocks()[0].max() == levels
        for _ in range(levels):
            lev, _ = m.get_blocks()
            assert m.adapt(np.where(lev == lev.max(), -1, 0).astype(np.int32))
            check()
        assert m.num_blocks == 2 ** dim
    m.close()


@pytest.mark.parametrize("poison", ["nan", "rho<=0", "p<=0"])
def test_invalid_cell_is_reported_by_compute_dt(poison):
    """A state with a NaN, a non-positive density or a non-positive pressure in ONE cell must not give a finite dt:
    both the stand-alone reduction and the maximum fused into the last stage report it (the oracle aborts on such a
    state, reading A18)."""
    cfg = W.config(3, scale=1)
    lm = f4.Mesh.from_config(cfg)
    lm.bind_torch()
    lev, co = lm.get_blocks()
    u = W.initial_state(cfg, lev, co)
    dt = None
    for fused in (False, True):
        lm.set_state(0, u)
        if fused:
            dt = lm.compute_dt(0, cfg["cfl"])
        bad = u.copy()
        if poison == "nan":
            bad[3, 4, 5, 6, 7] = np.nan
        elif poison == "rho<=0":
            bad[3, 0, 5, 6, 7] = -1.0
        else:
            bad[3, 4, 5, 6, 7] = 0.0          # E = 0 < kinetic energy: p < 0
        lm.set_state(0, bad)
        if fused:
            lm.advance(1e-3 * dt)             # the fused maximum of the new state sees the bad cell
        with pytest.raises(f4.F4Error):
            lm.compute_dt(0, cfg["cfl"])
    lm.close()


def test_asynchronous_regrid_matches_the_oracle_with_the_same_lag():
    """f4_adapt_begin / f4_adapt_end: the host part of the regrid runs on a worker thread while the device advances a
    step on the current mesh; the new mesh (the one f4_adapt builds from the same flags) takes over afterwards.  The
    oracle mirrors it -- flags at step s, advance, then adapt -- and the two runs agree to 1e-11."""
    cfg = dict(W.config(5), base_level=1, max_level=3)
    lm = f4.Mesh.from_config(cfg, max_blocks=3000)
    lm.bind_torch()
    om = O.OracleMesh.from_config(cfg)
    perm = _set_both(lm, om, cfg)
    om.fill_ghosts(0)
    fo, _ = om.refine_flags(0, om.CRIT_PJUMP, PJUMP)
    assert om.adapt(fo) == lm.adapt(fo[perm])
    perm = _set_both(lm, om, cfg)
    changed = 0
    for s in range(9):
        pend = None
        if s % 3 == 0:
            om.fill_ghosts(0)
            pend, _ = om.refine_flags(0, om.CRIT_PJUMP, PJUMP)
            lm.adapt_begin(pend[perm])
            with pytest.raises(f4.F4Error):
                lm.adapt(pend[perm])                   # no second regrid while one is pending
        dt = om.compute_dt(0, cfg["cfl"])
        assert abs(lm.compute_dt(0, cfg["cfl"]) - dt) <= 1e-12 * dt
        om.advance(dt)
        lm.advance(dt)
        if pend is not None:
            ch_g, ch_o = lm.adapt_end(), om.adapt(pend)
            assert ch_g == ch_o
            changed += ch_o
            perm = _perm(lm, om)
            assert np.all(H.rel_linf(lm.get_state(0), om.get_state(0)[perm]) <= TOL_STATE)
    assert changed >= 1 and lm.get_blocks()[0].max() == 3
    err = H.rel_linf(lm.get_state(0), om.get_state(0)[perm])
    assert np.all(err <= TOL_STATE), err
    with pytest.raises(f4.F4Error):
        lm.adapt_end()                                 # nothing pending
    lm.close()


@pytest.mark.parametrize("n,scale,flux_fix", [(1, None, False), (3, 1, False), (5, 1, False), (5, 1, True)])
def test_advance_cfl_equals_compute_dt_then_advance(n, scale, flux_fix):
    """f4_advance_cfl keeps dt on the device (no host round trip per step); it must be compute_dt followed by advance:
    bit-identical states and the same dt against a second mesh stepped the two-call way, and the oracle's state to 1e-11."""
    cfg = W.config(n, scale=scale)
    a = f4.Mesh.from_config(cfg, max_blocks=3000)
    b = f4.Mesh.from_config(cfg, max_blocks=3000)
    a.bind_torch()
    b.bind_torch()
    om = O.OracleMesh.from_config(cfg)
    if n == 5:
        fl = np.zeros(a.num_blocks, dtype=np.int32)
        fl[[0, 3, 5]] = 1
        perm0 = _perm(a, om)
        fo = np.empty_like(fl)
        fo[perm0] = fl
        assert a.adapt(fl) and b.adapt(fl) and om.adapt(fo)
        a.set_flux_fix(flux_fix)
        b.set_flux_fix(flux_fix)
        om.set_flux_fix(flux_fix)
    lev, co = a.get_blocks()
    u = W.initial_state(cfg, lev, co)
    a.set_state(0, u)
    b.set_state(0, u)
    perm = _perm(a, om)
    uo = np.empty_like(u)
    uo[perm] = u
    om.set_state(0, uo)
    for s in range(6):
        a.advance_cfl(cfg["cfl"])
        dt = b.compute_dt(0, cfg["cfl"])
        b.advance(dt)
        om.advance(om.compute_dt(0, cfg["cfl"]))
        if s in (0, 5):
            assert a.last_dt() == dt
    assert np.array_equal(a.get_state(0), b.get_state(0))
    err = H.rel_linf(a.get_state(0), om.get_state(0)[perm])
    assert np.all(err <= TOL_STATE), err
    a.close()
    b.close()


def test_advance_cfl_reports_an_invalid_state():
    cfg = W.config(3, scale=1)
    lm = f4.Mesh.from_config(cfg)
    lm.bind_torch()
    lev, co = lm.get_blocks()
    u = W.initial_state(cfg, lev, co)
    u[2, 0, 3, 3, 3] = -1.0
    lm.set_state(0, u)
    lm.advance_cfl(cfg["cfl"])              # runs with dt = 0 (and NaN fluxes around the bad cell)
    with pytest.raises(f4.F4Error):
        lm.last_dt()
    far = lm.get_state(0)[40:]              # blocks away from the bad cell: u + 0 * F(u) = u
    assert np.array_equal(far, u[40:])
    lm.close()

"""Pins for the CPU oracle (oracle/f4_oracle.cpp) against what the paper and
the mathematics fix -- SURVEY.md §8(c) pins P1..P11.  None of these compare
the oracle with itself or with the CUDA path."""
from __future__ import annotations

import os

import numpy as np
import pytest

import exact_riemann
import helpers as H
from oracle import oracle as O
from paper_2605_07612_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")
PER, OUT, KEEP = W.PERIODIC, W.OUTFLOW, W.KEEP


def _golden(name):
    rows = []
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                rows.append([float(x) for x in line.split()])
    return rows


def mesh(dim, N, brick, base, maxl, bc, gamma=1.4, ng=2):
    return O.OracleMesh(dim, N, ng, brick, base, maxl, bc, gamma, 2)


def run_steps(m, nsteps, cfl=0.4, dts=None):
    used = []
    for s in range(nsteps):
        dt = m.compute_dt(0, cfl) if dts is None else dts[s]
        m.advance(dt)
        used.append(dt)
    return used


# ---------------------------------------------------------------- elementary
def test_minmod_G_eq1():
    # PAPER.md:119-121 eq. (1)
    assert O.minmod_G(1.0, -2.0, 1.0) == 0.0
    assert O.minmod_G(-1.0, 2.0, 2.0) == 0.0
    assert O.minmod_G(0.0, 3.0, 1.0) == 0.0
    assert O.minmod_G(1.0, 3.0, 1.0) == 1.0          # min(|a|,|b|,|a+b|/2) = 1
    assert O.minmod_G(1.0, 3.0, 2.0) == 2.0          # min(2, 6, 2)
    assert O.minmod_G(1.0, 1.5, 2.0) == 1.25         # central difference wins
    assert O.minmod_G(-1.0, -3.0, 1.0) == -1.0
    assert O.minmod_G(-2.0, -0.5, 1.5) == -0.75
    for a in (0.3, 1.7, -2.2):
        assert O.minmod_G(a, a, 1.0) == a            # linear data: limiter inactive


def test_appendix_a_eq24():
    # lower fine child = 1 - 1/4 min(theta, M/2); golden thresholds
    M = 1e6
    for ndim, theta_max, v_at_max, v_at_1 in _golden("appendix_a.txt"):
        ndim = int(ndim)
        d1 = O.minmod_G(1.0 - 0.0, M - 1.0, 1.0)
        dm = O.minmod_G(1.0 - 0.0, M - 1.0, theta_max)
        assert 1.0 - ndim * 0.25 * d1 == v_at_1
        assert abs((1.0 - ndim * 0.25 * dm) - v_at_max) < 1e-15
        assert 1.0 - ndim * 0.25 * O.minmod_G(1.0, M - 1.0, theta_max * 1.01) < 0.0  # beyond threshold: negative


def test_vanleer_limiter():
    # reading A1: harmonic mean; symmetric, 0 at extrema, = a for linear data, bounded by 2 min(|a|,|b|)
    assert O.vanleer(1.0, -1.0) == 0.0 and O.vanleer(0.0, 1.0) == 0.0
    assert O.vanleer(2.0, 2.0) == 2.0
    assert O.vanleer(1.0, 3.0) == 1.5 and O.vanleer(3.0, 1.0) == 1.5
    assert O.vanleer(-1.0, -3.0) == -1.5
    rng = np.random.default_rng(0)
    for a, b in rng.uniform(0.01, 5, (50, 2)):
        s = O.vanleer(a, b)
        assert 0 < s <= 2 * min(a, b) + 1e-15
        assert abs(s - 2 * a * b / (a + b)) < 1e-15


def test_hll_flux_consistency_and_upwinding():
    g = 1.4
    # consistency: F(w,w) = physical flux, any direction (eq. 14)
    w = np.array([1.3, 0.4, -0.2, 0.7, 2.1])
    rho, u, p = w[0], w[1:4], w[4]
    E = p / (g - 1) + 0.5 * rho * u @ u
    for d in range(3):
        F = O.riemann_flux(3, g, w, w, d)
        ref = np.array([rho * u[d], *(rho * u * u[d] + p * np.eye(3)[d]), (E + p) * u[d]])
        assert np.allclose(F, ref, rtol=1e-14, atol=1e-15)
    # supersonic to the right: pure upwinding F = F(wL)
    wL = np.array([1.0, 5.0, 0.0, 0.0, 1.0])
    wR = np.array([0.9, 5.2, 0.1, 0.0, 0.8])
    F = O.riemann_flux(3, g, wL, wR, 0)
    EL = 1.0 / 0.4 + 0.5 * 25
    assert np.allclose(F, [5.0, 25 + 1.0, 0.0, 0.0, (EL + 1.0) * 5.0], rtol=1e-14)
    # Einfeldt speeds (reading A3) for equal states reduce to u -+ c (eq. 16)
    smin, smax = O.wavespeeds(3, g, w, w, 1)
    c = np.sqrt(g * p / rho)
    assert abs(smin - (u[1] - c)) < 1e-15 and abs(smax - (u[1] + c)) < 1e-15
    # mirror symmetry: swap L/R and negate the normal velocity -> mass flux changes sign exactly
    wLm, wRm = wR.copy(), wL.copy()
    wLm[1] *= -1
    wRm[1] *= -1
    Fm = O.riemann_flux(3, g, wLm, wRm, 0)
    Fo = O.riemann_flux(3, g, wL, wR, 0)
    assert Fm[0] == -Fo[0] and Fm[1] == Fo[1] and Fm[4] == -Fo[4]
    # Rusanov variant is consistent too
    assert np.allclose(O.riemann_flux(3, g, w, w, 2, O.FLUX_RUSANOV)[0], rho * u[2], rtol=1e-14)


def test_exact_riemann_solver_pinned():
    (ps, us), = _golden("sod_star.txt")
    p, u = exact_riemann.star_state((1, 0, 1), (0.125, 0, 0.1), 1.4)
    assert abs(p - ps) < 5e-5 and abs(u - us) < 5e-5


# ---------------------------------------------------------------- P1 uniform
@pytest.mark.parametrize("dim", [2, 3])
def test_P1_uniform_state_bit_exact(dim):
    # supersonic uniform state on an AMR mesh with outflow + periodic faces
    bc = [OUT, OUT, PER, PER, OUT, OUT][: 2 * dim]
    m = mesh(dim, 8, (2, 2, 2)[:dim], 0, 2, bc)
    flags = np.zeros(m.num_blocks, dtype=np.int32)
    flags[0] = 1
    assert m.adapt(flags)
    flags = np.zeros(m.num_blocks, dtype=np.int32)
    flags[3] = 1
    m.adapt(flags)
    lev, co = m.get_blocks()
    assert lev.max() >= 1
    cfg = dict(dim=dim, block_n=8, brick=(2, 2, 2), ic="uniform", rho0=1.7, vel0=(3.1, -0.4, 0.9), p0=0.6,
               gamma=1.4, seed=1)
    u0 = W.initial_state(cfg, lev, co)
    m.set_state(0, u0)
    run_steps(m, 4)
    assert np.array_equal(m.get_state(0), u0)


# ---------------------------------------------------------------- P2 conservation
@pytest.mark.parametrize("n", [1, 2])
def test_P2_conservation_periodic(n):
    cfg = W.config(n, scale=1 if n == 2 else None)
    m = O.OracleMesh.from_config(cfg)
    lev, co = m.get_blocks()
    m.set_state(0, W.initial_state(cfg, lev, co))
    t0 = m.totals(0)
    scale = np.abs(t0).max()
    for _ in range(5):
        run_steps(m, 1)
        t1 = m.totals(0)
        assert np.all(np.abs(t1 - t0) <= 1e-13 * scale), (t1 - t0) / scale


# ---------------------------------------------------------------- P3 Sod
def _sod_run(dim, axis, ncell, mirrored=False, dts=None, N=8):
    nb = ncell // N
    brick = [1, 1, 1]
    brick[axis] = nb
    bc = [PER] * 6
    bc[2 * axis] = bc[2 * axis + 1] = OUT
    m = mesh(dim, N, brick[:dim], 0, 0, bc[: 2 * dim])
    lev, co = m.get_blocks()
    cfg = dict(dim=dim, block_n=N, brick=tuple(brick))
    xyz, _ = W.cell_centres(cfg, lev, co)
    x = xyz[axis]
    left = x < 0.5
    if mirrored:
        left = ~left
    nvar = dim + 2
    w = np.zeros((len(lev), nvar) + x.shape[1:])
    w[:, 0] = np.where(left, 1.0, 0.125)
    w[:, nvar - 1] = np.where(left, 1.0, 0.1)
    m.set_state(0, W.prim_to_cons(w, 1.4))
    t, T, used = 0.0, 0.2, []
    k = 0
    while t < T:
        dt = m.compute_dt(0, 0.4) if dts is None else dts[k]
        if dts is None and t + dt > T:
            dt = T - t
        m.advance(dt)
        used.append(dt)
        t += dt
        k += 1
        if dts is not None and k == len(dts):
            break
    return m, x, used


def _profile(m, x, axis, dim):
    """1D profile along the tube + max transverse spread."""
    u = m.get_state(0)
    lev, co = m.get_blocks()
    order = np.argsort(co[:, axis])
    ax = 3 - axis  # array axis of [nb, z, y, x] after dropping var
    rho = np.moveaxis(u[order, 0], ax, 1)  # [nb, N, ...]
    xs = np.moveaxis(x[order], ax, 1)
    flat = rho.reshape(rho.shape[0] * rho.shape[1], -1)
    spread = np.abs(flat - flat[:, :1]).max()
    return xs.reshape(flat.shape[0], -1)[:, 0], flat[:, 0], spread, u[order]


def test_P3_sod_convergence_2d():
    errs = []
    for n in (128, 256, 512):
        m, x, _ = _sod_run(2, 0, n)
        xs, rho, spread, _ = _profile(m, x, 0, 2)
        assert spread == 0.0  # transverse direction stays exactly uniform
        ex, _, _ = exact_riemann.sample((1, 0, 1), (0.125, 0, 0.1), 1.4, (xs - 0.5) / 0.2)
        errs.append(np.mean(np.abs(rho - ex)))
    orders = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    # a 2nd-order TVD scheme is limited to < 1 by the smeared contact (0.7-1.0)
    assert errs[0] < 6e-3 and errs[2] < 2e-3, errs
    assert np.all(orders > 0.6) and np.all(orders < 1.1), (errs, orders)


def test_P3_sod_directions_and_mirror_3d():
    mx, x, dts = _sod_run(3, 0, 64)
    xs, rho_x, spread, _ = _profile(mx, x, 0, 3)
    assert spread == 0.0
    ex, _, _ = exact_riemann.sample((1, 0, 1), (0.125, 0, 0.1), 1.4, (xs - 0.5) / 0.2)
    assert np.mean(np.abs(rho_x - ex)) < 1.2e-2
    for axis in (1, 2):  # same dt sequence: profiles bit-identical along y and z
        ma, xa, _ = _sod_run(3, axis, 64, dts=dts)
        _, rho_a, spread_a, _ = _profile(ma, xa, axis, 3)
        assert spread_a == 0.0
        assert np.array_equal(rho_a, rho_x)
    mm, xm, _ = _sod_run(3, 0, 64, mirrored=True, dts=dts)
    _, rho_m, _, _ = _profile(mm, xm, 0, 3)
    assert np.array_equal(rho_m[::-1], rho_x)


# ---------------------------------------------------------------- P4 order of accuracy
def test_P4_density_wave_second_order():
    # u, p constant => Euler reduces to advection of rho; paper's finding for
    # van Leer + Heun: L1 order ~2, L2 order 1.7-1.8
    T = 0.2
    e1, e2 = [], []
    for lvl in (1, 2, 3):
        cfg = W.config(1, scale=lvl)
        m = O.OracleMesh.from_config(cfg)
        lev, co = m.get_blocks()
        m.set_state(0, W.initial_state(cfg, lev, co, noise=False))
        t = 0.0
        while t < T:
            dt = min(m.compute_dt(0, 0.4), T - t)
            m.advance(dt)
            t += dt
        (x, y), _ = W.cell_centres(cfg, lev, co)
        exact = 1.0 + 0.1 * np.sin(2 * np.pi * (x - 0.5 * T)) * np.sin(2 * np.pi * (y - 0.5 * T))
        d = m.get_state(0)[:, 0] - exact
        e1.append(np.mean(np.abs(d)))
        e2.append(np.sqrt(np.mean(d * d)))
    o1 = np.log2(np.array(e1[:-1]) / np.array(e1[1:]))
    o2 = np.log2(np.array(e2[:-1]) / np.array(e2[1:]))
    assert o1[-1] > 1.8 and o1[-1] < 2.3, (e1, o1)
    assert o2[-1] > 1.6 and o2[-1] < 1.9, (e2, o2)  # paper: 1.7-1.8


# ---------------------------------------------------------------- P5 linear field (paper's own test)
def _linear(X):
    phi = X[0] + 2.0 * X[1]
    if X.shape[0] == 3:
        phi = phi + 3.0 * X[2]
    return phi


def _set_boundary_ghosts(m, brick):
    lev, co = m.get_blocks()
    X, noncorner, outside = H.padded_coords(m.dim, m.N, m.Ng, brick, lev, co)
    phi = _linear(X)
    u = m.get_state(0, with_ghosts=True)
    for v in range(m.nvar):
        u[:, v] = np.where(outside, phi, u[:, v])
    m.set_state(0, u, with_ghosts=True)
    return phi, noncorner


def _check_linear(m, brick, tol):
    phi, noncorner = _set_boundary_ghosts(m, brick)
    m.fill_ghosts(0)
    u = m.get_state(0, with_ghosts=True)
    for v in range(m.nvar):
        err = np.abs(u[:, v] - phi)[noncorner].max()
        assert err <= tol, (v, err)


@pytest.mark.parametrize("dim,ng,nlev", [(2, 2, 4), (3, 2, 3), (2, 1, 3), (2, 3, 3), (2, 4, 3), (3, 1, 2), (3, 3, 2),
                                         (2, 2, 7), (3, 2, 5)])
def test_P5_linear_field(dim, ng, nlev):
    # PAPER.md:433-447 eq. (21)-(22): phi = x+2y+3z, refine around r_ref, fill, check incl. ghosts;
    # then remove the refinement one level at a time.  Paper's tolerance 1e-15 ("floating point
    # error"); we allow 4 ulp of max|phi| = 6 (3.6e-15): cell centres are rounded independently here.
    tol = 4 * np.spacing(6.0)
    brick = (2, 2, 2)[:dim]
    refs = [-1, 0, 1]
    pts = [(0.5 + 0.49 * i, 0.5 + 0.49 * j, 0.5 + 0.49 * k) for i in refs for j in refs for k in (refs if dim == 3 else [0])]
    if dim == 3 and nlev < 5:
        pts = pts[::2]  # 14 of the 27 points keep these cases short; corners, edges, faces and centre all occur
    # (2, 2, 7) and (3, 2, 5) are the paper's own extent: all 9 / 27 reference points, 7 / 5 levels
    for rref in pts:
        m = O.OracleMesh(dim, 8, ng, brick, 0, nlev, [KEEP] * (2 * dim), 1.4, 2)
        lev, co = m.get_blocks()
        X, _, _ = H.padded_coords(dim, 8, ng, brick, lev, co)
        u = m.get_state(0, with_ghosts=True)
        u[:] = _linear(X)[:, None]
        m.set_state(0, u, with_ghosts=True)
        _check_linear(m, brick, tol)
        for _ in range(nlev):  # add levels around r_ref
            lev, co = m.get_blocks()
            size = 1.0 / (2 * 2.0 ** lev)
            flags = np.ones(len(lev), dtype=np.int32)
            for a in range(dim):
                lo = co[:, a] * size
                flags &= ((lo <= rref[a]) & (rref[a] < lo + size)).astype(np.int32)
            assert flags.sum() == 1
            assert m.adapt(flags)
            lev, co = m.get_blocks()
            H.check_mesh_valid(dim, brick, [KEEP] * 6, lev, co, 0, nlev)
            _check_linear(m, brick, tol)
        assert m.get_blocks()[0].max() == nlev
        for _ in range(nlev):  # remove the refinement, one level per call
            lev, _ = m.get_blocks()
            flags = np.where(lev == lev.max(), -1, 0).astype(np.int32)
            assert m.adapt(flags)
            _check_linear(m, brick, tol)
        assert m.get_blocks()[0].max() == 0


# ---------------------------------------------------------------- P6 restriction
@pytest.mark.parametrize("dim", [2, 3])
def test_P6_restriction_is_block_average_and_roundtrip(dim):
    rng = np.random.default_rng(5)
    m = mesh(dim, 8, (2, 2, 2)[:dim], 0, 1, [PER] * (2 * dim))
    u0 = rng.uniform(0.5, 1.5, m.get_state(0).shape)
    m.set_state(0, u0)
    m.adapt(np.ones(m.num_blocks, dtype=np.int32))          # refine everything
    lev, co = m.get_blocks()
    assert (lev == 1).all()
    uf = m.get_state(0)
    # mean of the 2^d children of each coarse cell equals the parent to round-off (slopes cancel, A9)
    fine_sum = {}
    m2 = mesh(dim, 8, (2, 2, 2)[:dim], 0, 1, [PER] * (2 * dim))
    lev0, co0 = m2.get_blocks()
    k0 = H.key_index(lev0, co0)
    for b in range(len(lev)):
        par = k0[(0, co[b, 0] >> 1, co[b, 1] >> 1, co[b, 2] >> 1)]
        o = co[b] & 1
        blk = uf[b]
        if dim == 3:
            avg = blk.reshape(blk.shape[0], 4, 2, 4, 2, 4, 2).mean(axis=(2, 4, 6))
            ref = u0[par][:, o[2] * 4:(o[2] + 1) * 4, o[1] * 4:(o[1] + 1) * 4, o[0] * 4:(o[0] + 1) * 4]
        else:
            avg = blk.reshape(blk.shape[0], 1, 4, 2, 4, 2).mean(axis=(3, 5))
            ref = u0[par][:, :, o[1] * 4:(o[1] + 1) * 4, o[0] * 4:(o[0] + 1) * 4]
        assert np.abs(avg - ref).max() <= 4 * np.spacing(1.5)
    # coarsen back: restriction = exact block average in the pinned order (A8) -> bit-exact vs numpy pairwise
    m.adapt(-np.ones(m.num_blocks, dtype=np.int32))
    lev2, co2 = m.get_blocks()
    assert (lev2 == 0).all()
    uc = m.get_state(0)
    perm = H.match_blocks(lev2, co2, lev0, co0)
    assert np.abs(uc - u0[perm]).max() <= 4 * np.spacing(1.5)
    # bit-exact check of the coarse values against the pairwise x->y->z sum evaluated here
    kf = H.key_index(lev, co)
    for b in range(len(lev2)):
        for oz in range(2 if dim == 3 else 1):
            for oy in range(2):
                for ox in range(2):
                    f = uf[kf[(1, 2 * co2[b, 0] + ox, 2 * co2[b, 1] + oy, (2 * co2[b, 2] + oz) if dim == 3 else 0)]]
                    sx = f[..., 0::2] + f[..., 1::2]
                    sy = sx[..., 0::2, :] + sx[..., 1::2, :]
                    if dim == 3:
                        sz = (sy[:, 0::2] + sy[:, 1::2]) * 0.125
                        got = uc[b][:, oz * 4:(oz + 1) * 4, oy * 4:(oy + 1) * 4, ox * 4:(ox + 1) * 4]
                    else:
                        sz = sy * 0.25
                        got = uc[b][:, :, oy * 4:(oy + 1) * 4, ox * 4:(ox + 1) * 4]
                    assert np.array_equal(got, sz)


def test_P7_prolongation_closed_form_3d():
    # Appendix A in 3D through the regrid path: coarse values (0,1,M) along each axis around one cell
    M = 1e3
    for theta, expect in ((1.0, 0.25), (4.0 / 3.0, 0.0)):
        m = mesh(3, 8, (1, 1, 1), 0, 1, [PER] * 6)
        m.set_options(theta=theta)
        u = np.ones(m.get_state(0).shape)
        # cell (4,4,4) (0-based) = 1; its lower neighbours 0, upper neighbours M; others 1
        for a in range(3):
            lo = [4, 4, 4]
            hi = [4, 4, 4]
            lo[a] -= 1
            hi[a] += 1
            u[0, :, lo[2], lo[1], lo[0]] = 0.0
            u[0, :, hi[2], hi[1], hi[0]] = M
        m.set_state(0, u)
        m.adapt(np.ones(1, dtype=np.int32))
        lev, co = m.get_blocks()
        b = H.key_index(lev, co)[(1, 1, 1, 1)]       # child holding coarse cells 4..7
        uf = m.get_state(0)
        corner = uf[b, 0, 0, 0, 0]                   # lower-lower-lower child of coarse cell (4,4,4)
        assert abs(corner - expect) < 1e-15          # 1 - 3/4 theta
        assert uf[b, 0, 1, 1, 1] == 1.0 + 0.75 * theta


# ---------------------------------------------------------------- P8 permutation
def test_P8_block_permutation():
    cfg = dict(W.config(2, scale=1), max_level=2)
    rng = np.random.default_rng(3)
    res = []
    for shuffle in (False, True):
        m = O.OracleMesh.from_config(cfg)
        flags = np.zeros(m.num_blocks, dtype=np.int32)
        flags[5] = 1
        m.adapt(flags)
        if shuffle:
            m.permute(rng.permutation(m.num_blocks))
        lev, co = m.get_blocks()
        m.set_state(0, W.initial_state(cfg, lev, co))
        run_steps(m, 3, dts=[2e-3] * 3)
        res.append((lev, co, m.get_state(0)))
    perm = H.match_blocks(res[0][0], res[0][1], res[1][0], res[1][1])
    assert not np.array_equal(perm, np.arange(len(perm)))
    assert np.array_equal(res[0][2], res[1][2][perm])


# ---------------------------------------------------------------- P9 RK closed form
def test_P9_heun_closed_form():
    # eq. (6)-(7) with F(u) = lambda u: one step = (1 + z + z^2/2) u
    m = mesh(2, 8, (1, 1), 0, 0, [PER] * 4)
    rng = np.random.default_rng(1)
    u0 = rng.uniform(1, 2, m.get_state(0).shape)
    m.set_state(0, u0)
    lam, dt = -3.0, 0.05
    m.set_test_rhs(True, lam)
    m.advance(dt)
    z = lam * dt
    assert np.allclose(m.get_state(0), (1 + z + z * z / 2) * u0, rtol=1e-15, atol=0)
    # generic eq. (5) sub-step with weights
    m.set_state(0, u0)
    m.set_state(1, 2 * u0)
    m.forward_euler(1, 0, 0.1, [0.25, 0.75], [0, 1])
    assert np.allclose(m.get_state(1), 0.1 * lam * u0 + 0.25 * u0 + 0.75 * 2 * u0, rtol=1e-15)


@pytest.mark.parametrize("scheme,coef", [
    ("RK_EULER", [1, 1]), ("RK_HEUN", [1, 1, 1 / 2]), ("RK_SSP33", [1, 1, 1 / 2, 1 / 6]),
    ("RK_SSP43", [1, 1, 1 / 2, 1 / 6, 1 / 48]), ("RK_RK4", [1, 1, 1 / 2, 1 / 6, 1 / 24])])
def test_P9_rk_schemes_stability_polynomials(scheme, coef):
    # eq. (5)-(11) with F(u) = lambda u: one step multiplies u by the scheme's stability polynomial R(z), z = lambda dt
    # (textbook: Taylor polynomial of the scheme's order; SSPRK(4,3): (1 + z/2)(2/3 + (1 + z/2)^3 / 3)
    #  = 1 + z + z^2/2 + z^3/6 + z^4/48; RK4 eq. (8)-(11): sum_{k<=4} z^k / k!)
    m = O.OracleMesh(2, 8, 2, (1, 1), 0, 0, [PER] * 4, 1.4, 4)
    rng = np.random.default_rng(1)
    u0 = rng.uniform(1, 2, m.get_state(0).shape)
    for lam, dt in [(-3.0, 0.05), (0.7, 0.3), (-1.0, 1.0)]:
        m.set_state(0, u0)
        m.set_test_rhs(True, lam)
        m.advance(dt, getattr(m, scheme))
        z = lam * dt
        R = sum(c * z ** k for k, c in enumerate(coef))
        assert np.allclose(m.get_state(0), R * u0, rtol=4e-15, atol=0), scheme


@pytest.mark.parametrize("scheme", ["RK_EULER", "RK_SSP33", "RK_SSP43", "RK_RK4"])
def test_rk_schemes_uniform_state_conservation_and_order(scheme):
    cfg = W.config(1)
    # P1: a uniform state is a fixed point of every sub-step, bit for bit
    m = O.OracleMesh.from_config(cfg, n_states=4)
    lev, co = m.get_blocks()
    cu = dict(cfg, ic="uniform", rho0=1.3, vel0=(0.4, -0.2, 0.0), p0=0.9)
    u = W.initial_state(cu, lev, co)
    m.set_state(0, u)
    for _ in range(2):
        m.advance(1e-2, getattr(m, scheme))
    assert np.array_equal(m.get_state(0), u)
    # P2: conservative on a periodic mesh to round-off
    m.set_state(0, W.initial_state(cfg, lev, co))
    t0 = m.totals(0)
    for _ in range(3):
        m.advance(m.compute_dt(0, 0.4), getattr(m, scheme))
    assert np.all(np.abs(m.totals(0) - t0) <= 1e-13 * np.abs(t0).max())
    # temporal order: against a run with dt/8 of the same scheme on the same mesh (the spatial operator is the
    # same, so the difference is the time-integration error): halving dt divides it by ~2^order
    order = {"RK_EULER": 1, "RK_SSP33": 3, "RK_SSP43": 3, "RK_RK4": 4}[scheme]
    u0 = W.initial_state(cfg, lev, co, False)
    T = 0.04
    def run(nsteps):
        m.set_state(0, u0)
        for _ in range(nsteps):
            m.advance(T / nsteps, getattr(m, scheme))
        return m.get_state(0)
    ref = run(64)
    e1 = np.abs(run(4) - ref).max()
    e2 = np.abs(run(8) - ref).max()
    obs = np.log2(e1 / e2)
    assert obs > order - 0.6, (scheme, obs, e1, e2)


# ---------------------------------------------------------------- P10
def test_P10_lower_dimensional_data():
    # z-independent 3D data stays z-independent bit-exactly and equals the 2D code to round-off
    cfg2 = W.config(1)
    m2 = O.OracleMesh.from_config(cfg2)
    lev2, co2 = m2.get_blocks()
    u2 = W.initial_state(cfg2, lev2, co2)
    m2.set_state(0, u2)
    dts = run_steps(m2, 3)
    cfg3 = dict(cfg2, dim=3, brick=(2, 2, 1), base_level=1, max_level=1, bc=[PER] * 6)
    # brick (2,2,1) at level 1 -> 4x4x2 blocks; domain z-extent 1/2
    m3 = O.OracleMesh.from_config(cfg3)
    lev3, co3 = m3.get_blocks()
    k2 = H.key_index(lev2, co2)
    u3 = np.zeros(m3.get_state(0).shape)
    for b in range(len(lev3)):
        src = u2[k2[(1, co3[b, 0], co3[b, 1], 0)]]  # [4,1,8,8]
        u3[b, 0] = src[0]
        u3[b, 1] = src[1]
        u3[b, 2] = src[2]
        u3[b, 4] = src[3]
    m3.set_state(0, u3)
    run_steps(m3, 3, dts=dts)
    r3 = m3.get_state(0)
    assert np.array_equal(r3, np.broadcast_to(r3[:, :, :1], r3.shape))  # z-independent, bit-exact
    assert np.all(r3[:, 3] == 0.0)
    r2 = m2.get_state(0)
    for b in range(len(lev3)):
        src = r2[k2[(1, co3[b, 0], co3[b, 1], 0)]]
        got = r3[b][[0, 1, 2, 4], 0]
        assert np.abs(got - src[:, 0]).max() <= 1e-14


# ---------------------------------------------------------------- P11
def test_P11_mirror_symmetry_blast():
    cfg = dict(W.config(5, scale=0), base_level=1, max_level=1)
    m = O.OracleMesh.from_config(cfg)
    lev, co = m.get_blocks()
    (x, y, z), _ = W.cell_centres(cfg, lev, co)
    r2 = (x - 0.5) ** 2 + (y - 0.5) ** 2 + (z - 0.5) ** 2
    w = np.zeros((len(lev), 5) + x.shape[1:])
    w[:, 0] = 1.0
    w[:, 4] = np.where(r2 < 0.2 ** 2, 10.0, 0.1)
    m.set_state(0, W.prim_to_cons(w, 1.4))
    run_steps(m, 4)
    u = m.get_state(0)
    k = H.key_index(lev, co)
    ext = 2
    for b in range(len(lev)):
        bm = k[(1, ext - 1 - co[b, 0], co[b, 1], co[b, 2])]
        mir = u[bm][:, :, :, ::-1]
        assert np.abs(u[b, 0] - mir[0]).max() <= 1e-12 * np.abs(u[:, 0]).max()
        assert np.abs(u[b, 1] + mir[1]).max() <= 1e-12 * max(np.abs(u[:, 1]).max(), 1.0)
        assert np.abs(u[b, 4] - mir[4]).max() <= 1e-12 * np.abs(u[:, 4]).max()


# ---------------------------------------------------------------- mesh rules
def test_adapt_rules_and_balance_bruteforce():
    rng = np.random.default_rng(11)
    for dim in (2, 3):
        bc = ([PER, PER, OUT, OUT, PER, PER])[: 2 * dim]
        brick = (2, 1, 2)[:dim]
        m = mesh(dim, 8, brick, 1, 4, bc)
        for it in range(6):
            nb = m.num_blocks
            flags = rng.choice([-1, 0, 1], size=nb, p=[0.5, 0.35, 0.15]).astype(np.int32)
            lev_old, co_old = m.get_blocks()
            m.adapt(flags)
            lev, co = m.get_blocks()
            H.check_mesh_valid(dim, list(brick) + [1], bc + [PER] * (6 - len(bc)), lev, co, 1, 4)
            knew = H.key_index(lev, co)
            for b in range(nb):
                key = (int(lev_old[b]), *map(int, co_old[b]))
                if flags[b] > 0 and lev_old[b] < 4:
                    assert key not in knew                                  # refined blocks are gone
                if flags[b] >= 0:
                    par = (key[0] - 1, key[1] >> 1, key[2] >> 1, key[3] >> 1)
                    assert par not in knew                                  # never coarsened without consent
    # no change -> adapt reports unchanged (mesh revision)
    m = mesh(2, 8, (2, 2), 1, 3, [PER] * 4)
    assert not m.adapt(np.zeros(m.num_blocks, dtype=np.int32))
    assert not m.adapt(-np.ones(m.num_blocks, dtype=np.int32))          # already at base level


# ---------------------------------------------------------------- pins of the readings' implementations
def test_einfeldt_speeds_worked_value():
    # reading A3 by hand: rho_L=1, rho_R=4 -> r=(1,2); u=(0,3); p=(1,4) -> c^2 = gamma both sides;
    # u^ = 6/3 = 2; d^2 = (1*g + 2*g)/3 + 1/2 * 2/9 * 9 = g + 1
    g = 1.4
    smin, smax = O.wavespeeds(3, g, [1.0, 0.0, 7.0, -2.0, 1.0], [4.0, 3.0, 1.0, 5.0, 4.0], 0)
    assert abs(smin - (2.0 - np.sqrt(g + 1.0))) < 1e-15 and abs(smax - (2.0 + np.sqrt(g + 1.0))) < 1e-15


def test_rusanov_flux_worked_value():
    # reading A2 by hand on the states of the Einfeldt pin: S_min = 2 - sqrt(g+1), S_max = 2 + sqrt(g+1),
    # S = max(|S_min|, |S_max|) = 2 + sqrt(2.4) (a min-for-max slip gives 0.45 instead of 3.55);
    # U_L = (1, 0, 7, -2, 29), F_L = (0, 1, 0, 0, 0);  U_R = (4, 12, 4, 20, 80), F_R = (12, 40, 12, 60, 252);
    # F = (F_L + F_R)/2 - S/2 (U_R - U_L)
    g = 1.4
    S = 2.0 + np.sqrt(2.4)
    F = O.riemann_flux(3, g, [1.0, 0.0, 7.0, -2.0, 1.0], [4.0, 3.0, 1.0, 5.0, 4.0], 0, O.FLUX_RUSANOV)
    hand = np.array([6.0 - 1.5 * S, 20.5 - 6.0 * S, 6.0 + 1.5 * S, 30.0 - 11.0 * S, 126.0 - 25.5 * S])
    assert np.allclose(F, hand, rtol=1e-14, atol=1e-13), (F, hand)
    # and the HLL flux of the same states differs (S- = min(S_min, 0) = 0.45.. is not -S)
    assert not np.allclose(O.riemann_flux(3, g, [1.0, 0.0, 7.0, -2.0, 1.0], [4.0, 3.0, 1.0, 5.0, 4.0], 0), hand, rtol=1e-3)


def test_conversions_worked_value():
    # eq. (15) by hand, numbers written here: rho=2, u=(3,-4,12) (|u|^2 = 169), p=1.2, gamma=1.4
    #   E = p/(gamma-1) + rho |u|^2 / 2 = 3 + 169 = 172;  U = (2, 6, -8, 24, 172)
    U = O.to_conservative(3, 1.4, [2.0, 3.0, -4.0, 12.0, 1.2])
    assert np.allclose(U, [2.0, 6.0, -8.0, 24.0, 172.0], rtol=1e-15)
    w = O.to_primitive(3, 1.4, [2.0, 6.0, -8.0, 24.0, 172.0])
    assert np.allclose(w, [2.0, 3.0, -4.0, 12.0, 1.2], rtol=1e-13)
    # 2D: rho=0.5, u=(-2, 1), p=0.3, gamma=5/3: E = 0.3/(2/3) + 0.25*5 = 0.45 + 1.25 = 1.7
    U2 = O.to_conservative(2, 5.0 / 3.0, [0.5, -2.0, 1.0, 0.3])
    assert np.allclose(U2, [0.5, -1.0, 0.5, 1.7], rtol=1e-15)
    assert np.allclose(O.to_primitive(2, 5.0 / 3.0, U2), [0.5, -2.0, 1.0, 0.3], rtol=1e-14)


def test_block_parallel_driver_is_bit_identical():
    # the all-cores timing leg of bench.py runs the unchanged routines over block ranges on several threads
    cfg = W.config(5, scale=1)
    a, b = O.OracleMesh.from_config(cfg), O.OracleMesh.from_config(cfg)
    f = np.zeros(a.num_blocks, dtype=np.int32)
    f[[0, 77, 300]] = 1
    assert a.adapt(f) and b.adapt(f)
    lev, co = a.get_blocks()
    u = W.initial_state(cfg, lev, co)
    a.set_state(0, u)
    b.set_state(0, u)
    for nthreads in (3, 5):
        dta, dtb = a.compute_dt(0, 0.4), b.compute_dt_mt(0, 0.4, nthreads)
        assert dta == dtb
        a.advance(dta)
        b.advance_mt(dtb, nthreads)
        assert np.array_equal(a.get_state(0, with_ghosts=True), b.get_state(0, with_ghosts=True))


def test_cfl_rate_uniform_closed_form():
    # reading A5: sum over dimensions of (|u_d| + c)/dx; uniform state u=(3,-4,0), rho=2, p=10/7 -> c=1
    cfg = dict(dim=3, block_n=8, brick=(2, 2, 2), ic="uniform", rho0=2.0, vel0=(3.0, -4.0, 0.0), p0=10.0 / 7.0,
               gamma=1.4, seed=1)
    m = mesh(3, 8, (2, 2, 2), 0, 0, [PER] * 6)
    lev, co = m.get_blocks()
    m.set_state(0, W.initial_state(cfg, lev, co))
    dx = 1.0 / 16
    assert abs(m.max_wave_rate(0) - (3 + 4 + 0 + 3 * 1.0) / dx) < 1e-12 * 160
    assert abs(m.compute_dt(0, 0.4) - 0.4 * dx / 10.0) < 1e-16
    # AMR: the finest level sets the rate (one global dt)
    m = mesh(3, 8, (2, 2, 2), 0, 1, [PER] * 6)
    f = np.zeros(8, dtype=np.int32)
    f[2] = 1
    m.adapt(f)
    lev, co = m.get_blocks()
    m.set_state(0, W.initial_state(cfg, lev, co))
    assert abs(m.max_wave_rate(0) - 10.0 / (dx / 2)) < 1e-12 * 320


@pytest.mark.parametrize("dim", [2, 3])
def test_srl_and_outflow_ghosts_by_definition(dim):
    # a1: ghost = the periodic neighbour's cell; a2 / reading A10: outflow ghost = nearest interior layer.
    # Field = unique integer per (var, global cell), so any index slip shows.
    N, ng = 8, 2
    brick = (3, 2, 2)[:dim]
    bc = [PER, PER, OUT, OUT, PER, PER][: 2 * dim]
    m = mesh(dim, N, brick, 0, 0, bc)
    lev, co = m.get_blocks()
    ext = [brick[a] * N for a in range(dim)] + ([1] if dim == 2 else [])

    def field(v, gi, gj, gk):
        return (((v * 1000.0 + gk) * 1000.0 + gj) * 1000.0 + gi)

    idx = np.arange(-ng, N + ng)
    u = np.zeros(m.get_state(0).shape)
    ar = np.arange(N)
    for b in range(len(lev)):
        gi = co[b, 0] * N + ar
        gj = co[b, 1] * N + ar
        gk = (co[b, 2] * N + ar) if dim == 3 else np.zeros(1, dtype=int)
        for v in range(m.nvar):
            u[b, v] = field(v, gi[None, None, :], gj[None, :, None], gk[:, None, None])
    m.set_state(0, u)
    m.fill_ghosts(0)
    p = m.get_state(0, with_ghosts=True)
    for b in range(len(lev)):
        gi = co[b, 0] * N + idx
        gj = co[b, 1] * N + idx
        gk = (co[b, 2] * N + idx) if dim == 3 else np.zeros(1, dtype=int)
        gi = np.mod(gi, ext[0])                                   # periodic in x
        gj = np.clip(gj, 0, ext[1] - 1)                           # outflow in y: clamp = nearest interior
        if dim == 3:
            gk = np.mod(gk, ext[2])
        GI, GJ, GK = gi[None, None, :], gj[None, :, None], gk[:, None, None]
        out = ((idx < 0) | (idx >= N)).astype(int)
        nout = out[None, None, :] + out[None, :, None] + (out[:, None, None] if dim == 3 else 0)
        for v in range(m.nvar):
            ref = field(v, GI, GJ, GK) * np.ones(p[b, v].shape)
            assert np.array_equal(p[b, v][nout <= 1], ref[nout <= 1])


# ---------------------------------------------------------------- flux fixing (test of 403-409)
def _amr_periodic_wave(dim, N=8):
    """Static refinement on a periodic mesh (the paper's flux-fixing test, with Euler instead of
    scalar advection): smooth density / pressure wave moving diagonally across the refinement boundaries."""
    cfg = dict(dim=dim, block_n=N, n_ghost=2, brick=(2, 2, 2)[:dim] + (1,) * (3 - dim), base_level=1, max_level=2,
               bc=[PER] * 6, gamma=1.4, seed=77, ic="uniform")
    m = O.OracleMesh.from_config(cfg)
    lev, co = m.get_blocks()
    flags = np.zeros(len(lev), dtype=np.int32)
    for b, c in enumerate(co):
        if all(1 <= c[a] <= 2 for a in range(dim)):
            flags[b] = 1
    assert m.adapt(flags)
    lev, co = m.get_blocks()
    assert lev.min() == 1 and lev.max() == 2
    xyz, _ = W.cell_centres(cfg, lev, co)
    w = np.zeros((len(lev), dim + 2) + xyz[0].shape[1:])
    ph = sum(xyz)
    w[:, 0] = 1.0 + 0.2 * np.sin(2 * np.pi * ph)
    for a in range(dim):
        w[:, 1 + a] = 0.7 + 0.1 * a
    w[:, dim + 1] = 1.0 + 0.1 * np.cos(2 * np.pi * xyz[0])
    m.set_state(0, np.ascontiguousarray(W.prim_to_cons(w, 1.4)))
    return m


@pytest.mark.parametrize("dim", [2, 3])
def test_flux_fixing_restores_conservation_on_static_refinement(dim):
    # the paper's e_cons, eq. (18): "on the order of machine precision" with flux fixing; without it the
    # coarse and fine fluxes at refinement boundaries differ and the totals drift
    drift = {}
    for fix in (False, True):
        m = _amr_periodic_wave(dim)
        m.set_flux_fix(fix)
        t0 = m.totals(0)
        run_steps(m, 6 if dim == 2 else 3)
        drift[fix] = np.abs(m.totals(0) - t0).max() / np.abs(t0).max()
    assert drift[True] <= 5e-15, drift
    assert drift[False] >= 1e-9, drift      # the test is able to see a missing correction


def test_flux_fixing_is_a_no_op_on_uniform_meshes_and_keeps_uniform_states():
    cfg = W.config(1)
    a, b = O.OracleMesh.from_config(cfg), O.OracleMesh.from_config(cfg)
    b.set_flux_fix(True)
    lev, co = a.get_blocks()
    u = W.initial_state(cfg, lev, co)
    a.set_state(0, u), b.set_state(0, u)
    dts = run_steps(a, 3)
    run_steps(b, 3, dts=dts)
    assert np.array_equal(a.get_state(0), b.get_state(0))
    # P1 with refinement boundaries: Fc == Ff for a constant state, so the correction is exactly zero
    m = _amr_periodic_wave(2)
    lev, co = m.get_blocks()
    cu = dict(dim=2, block_n=8, n_ghost=2, brick=(2, 2, 1), ic="uniform", rho0=1.3, vel0=(0.4, -0.2, 0.0), p0=0.9,
              gamma=1.4, seed=1)
    u = W.initial_state(cu, lev, co)
    m.set_flux_fix(True)
    m.set_state(0, u)
    run_steps(m, 3)
    assert np.array_equal(m.get_state(0), u)


# ---------------------------------------------------------------- refinement criteria (eq. 12; A15)
LOHNER = (5e-2, 6.25e-3, 1e-2, 1e-10)     # c_refine, c_derefine, eps, eps_abs of PAPER.md:560


def _one_block(dim, N=8, bc=KEEP):
    return mesh(dim, N, (1,) * dim, 0, 0, [bc] * (2 * dim))


def _padded_from_profile(dim, N, prof_x, var=0, base=0.0):
    """Natural padded state [1, nvar, Pz, P, P] whose variable `var` depends on x only: prof_x[P] (ghosts included)."""
    P = N + 4
    u = np.full((1, dim + 2, P if dim == 3 else 1, P, P), base)
    u[0, var] = np.asarray(prof_x)[None, None, :]
    return u


@pytest.mark.parametrize("dim", [2, 3])
def test_lohner_indicator_hand_values(dim):
    # one triple at cells (3,4,5) of an otherwise constant row: the block indicator is the largest E of the cells
    # whose stencil sees the triple; the golden file holds numerator and denominator worked by hand
    N, P = 8, 12
    for um, u0, up, num, den in _golden("lohner_eq12.txt"):
        m = _one_block(dim, N)
        prof = np.empty(P)
        prof[:5] = um            # padded index p = i + 1 (1-based interior i): cells <= 3 hold um
        prof[5] = u0             # cell 4
        prof[6:] = up            # cells >= 5
        m.set_state(0, _padded_from_profile(dim, N, prof), with_ghosts=True)
        flags, ind = m.refine_flags(0, m.CRIT_LOHNER, LOHNER)
        # stencils centred on cells 3 and 5 see (um,um,u0) and (u0,up,up): include them in the expectation
        def E(a, b, c):
            return abs(a - 2 * b + c) / (1e-10 + abs(b - a) + abs(c - b) + 1e-2 * (abs(a) + 2 * abs(b) + abs(c)))
        centre = num / (den + 1e-10)
        assert abs(E(um, u0, up) - centre) <= 1e-15            # the hand-worked row is what the formula gives
        expect = max(centre, E(um, um, u0), E(u0, up, up))
        assert abs(ind[0] - expect) <= 2e-16 * max(expect, 1.0), (um, u0, up, ind[0], expect)
        assert flags[0] == (1 if expect > LOHNER[0] else (-1 if expect < LOHNER[1] else 0))


def test_lohner_linear_field_is_never_refined_and_norm_is_euclidean():
    # a linear field has zero second differences: |E| = 0 in every cell -> derefine (the paper's linear-field
    # test input, eq. 21); a step in x, y and z at the same cell gives |E| = sqrt(3) E_1
    dim, N, P = 3, 8, 12
    m = _one_block(dim, N)
    idx = np.arange(P, dtype=np.float64)
    u = np.zeros((1, 5, P, P, P))
    u[0, 0] = 1.0 * idx[None, None, :] + 2.0 * idx[None, :, None] + 3.0 * idx[:, None, None]
    m.set_state(0, u, with_ghosts=True)
    flags, ind = m.refine_flags(0, m.CRIT_LOHNER, LOHNER)
    assert ind[0] == 0.0 and flags[0] == -1
    step = (idx >= 6).astype(np.float64)                       # cells <= 4 are 0, cells >= 5 are 1
    u[0, 0] = step[None, None, :] + step[None, :, None] + step[:, None, None]
    m.set_state(0, u, with_ghosts=True)
    _, ind3 = m.refine_flags(0, m.CRIT_LOHNER, (5e-2, 6.25e-3, 0.0, 0.0))
    # eps = eps_abs = 0: at cell (4,4,4) every direction sees (0,0,1) -> E_n = 1, |E| = sqrt(3); no cell exceeds it
    assert abs(ind3[0] - np.sqrt(3.0)) <= 4e-16


def test_lohner_scale_invariance_thresholds_and_ghost_use():
    dim, N, P = 2, 8, 12
    rng = np.random.default_rng(5)
    base = rng.uniform(0.5, 2.0, (1, 4, 1, P, P))
    m = _one_block(dim, N)
    m.set_state(0, base, with_ghosts=True)
    _, i1 = m.refine_flags(0, m.CRIT_LOHNER, (5e-2, 6.25e-3, 1e-2, 0.0), var=2)
    m.set_state(0, 1024.0 * base, with_ghosts=True)            # eps_abs = 0: E is homogeneous of degree 0
    _, i2 = m.refine_flags(0, m.CRIT_LOHNER, (5e-2, 6.25e-3, 1e-2, 0.0), var=2)
    assert i1[0] == i2[0] and i1[0] > 0
    # strict comparisons (reading A19): thresholds equal to the indicator keep the block
    for cr, cd, want in [(i1[0], 0.0, 0), (np.nextafter(i1[0], 0), 0.0, 1), (9.0, i1[0], 0), (9.0, np.nextafter(i1[0], 9), -1)]:
        f, _ = m.refine_flags(0, m.CRIT_LOHNER, (cr, cd, 1e-2, 0.0), var=2)
        assert f[0] == want
    # only face ghosts of the first layer are read: a spike in the first ghost layer is seen, one in the second
    # layer or in a corner ghost is not ("we do not consider cross-derivative terms")
    flat = np.ones((1, 4, 1, P, P))
    for (jj, ii), seen in [((5, 1), True), ((5, 0), False), ((1, 1), False), ((10, 6), True), ((11, 6), False)]:
        u = flat.copy()
        u[0, 0, 0, jj, ii] = 2.0
        m.set_state(0, u, with_ghosts=True)
        _, ind = m.refine_flags(0, m.CRIT_LOHNER, LOHNER)
        assert (ind[0] > 0) == seen, (jj, ii)


def test_pressure_jump_rule_hand_values_and_harness_definition():
    # reading A15: J = max |pa - pb| / min(pa, pb) over face-adjacent pairs, interior + first ghost layer
    cfg = dict(dim=3, block_n=8, n_ghost=2, brick=(2, 1, 1), base_level=0, max_level=0, bc=[PER] * 6, gamma=1.4)
    m = O.OracleMesh.from_config(cfg)
    lev, co = m.get_blocks()
    w = np.zeros((2, 5, 8, 8, 8))
    w[:, 0] = 1.0
    w[:, 4] = 0.7
    b0 = int(np.argmax(co[:, 0] == 0))
    def flags_for(cell, factor):
        ww = w.copy()
        ww[(b0, 4) + cell] = 0.7 * factor
        m.set_state(0, np.ascontiguousarray(W.prim_to_cons(ww, 1.4)))
        m.fill_ghosts(0)
        return m.refine_flags(0, m.CRIT_PJUMP, (0.1, 0.025))
    f, J = flags_for((3, 3, 3), 1.0)
    assert np.all(J == 0.0) and np.all(f == -1)                # uniform pressure
    f, J = flags_for((3, 3, 3), 2.0)                           # interior cell: only its own block sees it
    assert abs(J[b0] - 1.0) <= 1e-15 and f[b0] == 1 and J[1 - b0] == 0.0 and f[1 - b0] == -1
    f, J = flags_for((3, 3, 7), 0.5)                           # cell at the +x face: the neighbour sees it in its ghost
    assert abs(J[b0] - 1.0) <= 1e-15 and abs(J[1 - b0] - 1.0) <= 1e-15 and np.all(f == 1)
    f, J = flags_for((3, 3, 3), 1.05)                          # 0.025 < 0.05 < 0.1: keep
    assert abs(J[b0] - 0.05) <= 1e-14 and f[b0] == 0
    # the harness's numpy statement of the same rule (tests/helpers.py), on a config-5 blast with refinement
    cfg5 = W.config(5, scale=1)
    m5 = O.OracleMesh.from_config(cfg5)
    for _ in range(2):
        l5, c5 = m5.get_blocks()
        m5.set_state(0, W.initial_state(cfg5, l5, c5))
        m5.fill_ghosts(0)
        f5, _ = m5.refine_flags(0, m5.CRIT_PJUMP, (0.1, 0.025))
        assert np.array_equal(f5, H.pressure_jump_flags_numpy(cfg5, m5.get_state(0, with_ghosts=True)))
        assert (f5 == 1).any() and (f5 == -1).any()
        m5.adapt(f5)


# ---------------------------------------------------------------- gravity source term, eq. (20)
@pytest.mark.parametrize("dim", [2, 3])
def test_gravity_source_free_fall_closed_form(dim):
    # a uniform gas in a periodic box under S = (0, rho g, rho g.u): the fluxes cancel exactly, so rho and p stay
    # constant, u(t) = u0 + g t and E(t) = E0 + rho (g.u0 t + g^2 t^2 / 2).  dE/dt is linear in t, which Heun's
    # trapezoidal rule integrates exactly: the discrete solution equals the closed form to round-off
    cfg = dict(dim=dim, block_n=8, n_ghost=2, brick=(2, 2, 1), base_level=0, max_level=0, bc=[PER] * 6, gamma=5.0 / 3.0)
    m = O.OracleMesh.from_config(cfg)
    lev, co = m.get_blocks()
    rho, p0 = 0.7, 1.3
    u0 = np.array([0.3, -0.2, 0.1][:dim])
    g = np.array([0.0, -1.0, 0.5][:dim]) if dim == 3 else np.array([0.25, -1.0])
    w = np.zeros(m.get_state(0).shape)
    w[:, 0] = rho
    for a in range(dim):
        w[:, 1 + a] = u0[a]
    w[:, dim + 1] = p0
    m.set_state(0, W.prim_to_cons(w, cfg["gamma"]))
    m.set_gravity(g)
    t, dt = 0.0, 0.01
    for _ in range(5):
        m.advance(dt)
        t += dt
    u = m.get_state(0)
    E0 = p0 / (cfg["gamma"] - 1) + 0.5 * rho * u0 @ u0
    assert np.abs(u[:, 0] - rho).max() == 0.0
    for a in range(dim):
        assert np.abs(u[:, 1 + a] - rho * (u0[a] + g[a] * t)).max() <= 4e-16
    assert np.abs(u[:, dim + 1] - (E0 + rho * (g @ u0 * t + 0.5 * g @ g * t * t))).max() <= 2e-15
    # g = 0 is bit-identical to the path without a source term
    a_, b_ = O.OracleMesh.from_config(W.config(1)), O.OracleMesh.from_config(W.config(1))
    l1, c1 = a_.get_blocks()
    ui = W.initial_state(W.config(1), l1, c1)
    a_.set_state(0, ui), b_.set_state(0, ui)
    b_.set_gravity((0.0, 0.0))
    dts = run_steps(a_, 2)
    run_steps(b_, 2, dts=dts)
    assert np.array_equal(a_.get_state(0), b_.get_state(0))


def test_gravity_hydrostatic_balance_converges_at_second_order():
    # isothermal atmosphere rho = p = exp(-y) (g = (0,-1), c_iso^2 = 1) is an exact steady state of the equations:
    # the discrete residual (velocity picked up in a short time) must fall ~4x per mesh doubling for a
    # second-order scheme; a wrong sign or a missing energy source does not converge at all
    errs = []
    for base in (1, 2, 3):
        cfg = dict(dim=2, block_n=8, n_ghost=2, brick=(1, 1, 1), base_level=base, max_level=base,
                   bc=[PER, PER, KEEP, KEEP], gamma=1.4, ic="uniform")
        m = O.OracleMesh.from_config(cfg)
        lev, co = m.get_blocks()
        X, nc, _ = H.padded_coords(2, 8, 2, (1, 1), lev, co)
        w = np.zeros((len(lev), 4) + X[0].shape[1:])
        w[:, 0] = np.exp(-X[1])
        w[:, 3] = np.exp(-X[1])
        m.set_state(0, W.prim_to_cons(w, 1.4), with_ghosts=True)     # analytic values in the KEEP boundary ghosts
        m.set_state(1, W.prim_to_cons(w, 1.4), with_ghosts=True)
        m.set_gravity((0.0, -1.0))
        T, n = 0.02, 2 ** base
        for _ in range(n):
            m.advance(T / n)
        u = m.get_state(0)
        errs.append(np.abs(u[:, 2] / u[:, 0]).max())
    assert errs[0] / errs[1] > 3.0 and errs[1] / errs[2] > 3.0, errs


# ---------------------------------------------------------------- uniform Dirichlet / Neumann boundaries
DIR, NEU = W.DIRICHLET, W.NEUMANN


@pytest.mark.parametrize("dim", [2, 3])
def test_dirichlet_and_neumann_ghosts_reproduce_a_linear_profile(dim):
    # u_v = a_v + b_v * n along the normal of the boundary, everything in binary fractions so that the expected
    # ghost values are exact: with u_b = the face value (Dirichlet) or u_b' = the outward derivative (Neumann) the
    # ghost cells must continue the linear profile (a wrong sign, layer index or mirror cell breaks it)
    N, P = 8, 12
    nvar = dim + 2
    a_v = np.array([1.0, -0.5, 0.25, 2.0, 3.0][:nvar])
    b_v = np.array([2.0, 1.0, -4.0, 0.5, -1.0][:nvar])
    dx = 1.0 / N
    for axis in range(dim):
        for kind in (DIR, NEU):
            bc = [PER] * 6
            bc[2 * axis] = bc[2 * axis + 1] = kind
            m = O.OracleMesh(dim, N, 2, (1,) * dim, 0, 0, bc, 1.4, 2)
            x = (np.arange(-2, N + 2) + 0.5) * dx                     # cell centres along the axis, ghosts included
            shape = [1, 1, 1]
            shape[2 - axis] = P
            prof = x.reshape(shape)
            u = np.zeros((1, nvar, P if dim == 3 else 1, P, P))
            for v in range(nvar):
                u[0, v] = a_v[v] + b_v[v] * prof
            vals = np.zeros((6, nvar))
            if kind == DIR:
                vals[2 * axis] = a_v                                   # face at x = 0
                vals[2 * axis + 1] = a_v + b_v                         # face at x = 1
            else:
                vals[2 * axis] = -b_v                                  # outward normal derivative
                vals[2 * axis + 1] = b_v
            m.set_bc_values(vals)
            interior = u[:, :, 2:-2, 2:-2, 2:-2] if dim == 3 else u[:, :, :, 2:-2, 2:-2]
            m.set_state(0, np.ascontiguousarray(interior))
            m.fill_ghosts(0)
            g = m.get_state(0, with_ghosts=True)
            sl = [slice(None), slice(None)] + ([slice(2, -2)] * 3 if dim == 3 else [slice(0, 1), slice(2, -2), slice(2, -2)])
            sl[4 - axis] = slice(None)                                 # all cells along the axis, interior transverse
            assert np.array_equal(g[tuple(sl)], u[tuple(sl)]), (axis, kind)


def test_neumann_zero_derivative_is_outflow_and_dirichlet_hand_value():
    cfg = dict(dim=2, block_n=8, n_ghost=2, brick=(2, 1, 1), base_level=0, max_level=0, gamma=1.4)
    rng = np.random.default_rng(3)
    a = O.OracleMesh.from_config(dict(cfg, bc=[OUT] * 6))
    b = O.OracleMesh.from_config(dict(cfg, bc=[NEU] * 6))
    c = O.OracleMesh.from_config(dict(cfg, bc=[DIR] * 6))
    u = rng.uniform(0.5, 2.0, a.get_state(0).shape)
    vals = np.arange(24, dtype=np.float64).reshape(6, 4) / 8.0
    for m in (a, b, c):
        m.set_state(0, u)
    b.set_bc_values(np.zeros((6, 4)))
    c.set_bc_values(vals)
    for m in (a, b, c):
        m.fill_ghosts(0)
    ga, gb, gc = (m.get_state(0, with_ghosts=True) for m in (a, b, c))
    assert np.array_equal(ga, gb)                                      # u_b' = 0: the outflow rule, bit for bit
    lev, co = c.get_blocks()
    b0 = int(np.argmax(co[:, 0] == 0))
    # -x face (direction 0) of the left block, variable 2, row j = 3 (padded 5): ghost layers 1, 2 mirror cells 1, 2
    for gl in (1, 2):
        assert gc[b0, 2, 0, 5, 2 - gl] == 2.0 * vals[0, 2] - u[b0, 2, 0, 3, gl - 1]
    # +y face (direction 3), variable 1, column i = 6 (padded 8)
    for gl in (1, 2):
        assert gc[b0, 1, 0, 9 + gl, 8] == 2.0 * vals[3, 1] - u[b0, 1, 0, 8 - gl, 6]


# ---------------------------------------------------------------- Koren and WENO3 reconstructions
def test_koren_and_weno3_elementary_values():
    # Koren: the third-order slope (a + 2b)/3 towards the b side, limited to [0, 2a] and [0, 2b] (reading A1b)
    assert O.koren(1.0, 1.0) == 1.0 and O.koren(-2.0, -2.0) == -2.0          # linear data: exact
    assert O.koren(1.0, -1.0) == 0.0 and O.koren(0.0, 3.0) == 0.0             # extremum: zero slope
    assert O.koren(1.0, 4.0) == 2.0                                            # min(2a, (a+2b)/3 = 3, 2b = 8) = 2a
    assert O.koren(4.0, 1.0) == 2.0                                            # min(8, 2, 2b = 2)
    assert abs(O.koren(1.0, 1.5) - 4.0 / 3.0) <= 2e-16                        # unlimited: (1 + 3)/3
    assert abs(O.koren(1.5, 1.0) - 3.5 / 3.0) <= 2e-16 and O.koren(1.5, 1.0) != O.koren(1.0, 1.5)   # not symmetric
    assert O.koren(-1.0, -1.5) == -O.koren(1.0, 1.5)
    # kappa = 1/3: for a quadratic the face value w + s/2 is third-order: u = x^2 at x = -1, 0, 1 -> u(1/2) = 1/4;
    # a = -1, b = 1 is an extremum (limited), so test on x = 1, 2, 3: a = 3, b = 5, exact u(2.5) = 6.25, cell values
    # being point values here the kappa-scheme gives 4 + (3 + 10)/6 = 6.1667 = the quadratic through CELL AVERAGES
    assert abs((4.0 + 0.5 * O.koren(3.0, 5.0)) - (4.0 + 13.0 / 6.0)) <= 1e-15
    # WENO3: smooth data -> the ideal weights 1/3, 2/3 -> the same (a + 2b)/3 up to O(differences of a, b)
    assert abs(O.weno3(0.5, 0.5) - 0.5) <= 1e-16
    assert abs(O.weno3(1e-3, 1.001e-3) - (1e-3 + 2 * 1.001e-3) / 3) <= 1e-9
    # a jump on one side: the stencil across it gets a vanishing weight (ENO property); value worked by hand:
    # a = 0, b = 1: alpha0 = (1/3)/eps^2, alpha1 = (2/3)/(1+eps)^2 -> s = alpha1 / (alpha0 + alpha1) ~ 2e-12
    al0, al1 = (1 / 3) / 1e-12, (2 / 3) / (1 + 1e-6) ** 2
    assert abs(O.weno3(0.0, 1.0) - al1 / (al0 + al1)) <= 1e-24 and O.weno3(0.0, 1.0) < 1e-11
    assert abs(O.weno3(1.0, 0.0) - al0 * 0 - ((1 / 3) / (1 + 1e-6) ** 2) / ((1 / 3) / (1 + 1e-6) ** 2 + (2 / 3) / 1e-12)) <= 1e-24


@pytest.mark.parametrize("limiter,name,min_order,max_ratio", [(O.LIM_KOREN, "koren", 2.0, 0.6), (O.LIM_WENO3, "weno3", 2.8, 0.4)])
def test_third_order_reconstructions_converge_faster_than_van_leer(limiter, name, min_order, max_ratio):
    # smooth density wave (exact solution = translation), SSPRK(3,3) at a small CFL number so that the spatial error
    # dominates.  van Leer gives L1 order ~1.95 here ("approximately 2"); the kappa = 1/3 slope of
    # Koren's limiter is third-order where the limiter is inactive but clips the extrema of the wave (observed
    # 2.1, half of van Leer's error); WENO3 does not clip and approaches its formal order 3 (observed 2.5 -> 3.8)
    def l1_error(lim, base):
        cfg = dict(W.config(1), base_level=base, max_level=base)
        m = O.OracleMesh.from_config(cfg, n_states=3)
        m.set_options(lim, O.FLUX_HLL, 1.0)
        lev, co = m.get_blocks()
        m.set_state(0, W.initial_state(cfg, lev, co, False))
        T, n = 0.1, 5 * 2 ** base
        for _ in range(n):
            m.advance(T / n, m.RK_SSP33)
        xyz, _ = W.cell_centres(cfg, lev, co)
        exact = 1.0 + 0.1 * np.sin(2 * np.pi * (xyz[0] - 0.5 * T)) * np.sin(2 * np.pi * (xyz[1] - 0.5 * T))
        return np.abs(m.get_state(0)[:, 0] - exact).mean()
    e = [l1_error(limiter, b) for b in (2, 3)]
    ev = l1_error(O.LIM_VANLEER, 3)
    order = np.log2(e[0] / e[1])
    assert order > min_order, (name, e, order)
    assert e[1] < max_ratio * ev, (name, e[1], ev)


@pytest.mark.parametrize("limiter", [O.LIM_KOREN, O.LIM_WENO3])
def test_asymmetric_reconstructions_keep_mirror_symmetry(limiter):
    # Koren / WENO3 slopes are not symmetric in (a, b): the right state of a cell's low face must use the slope
    # with the arguments exchanged.  Then a run and its mirror image (x -> 1 - x, u -> -u) stay mirror images to
    # round-off; using the same slope on both faces breaks this at the first step
    cfg = dict(W.config(1), base_level=1, max_level=1)
    outs = []
    for mirror in (False, True):
        m = O.OracleMesh.from_config(cfg)
        m.set_options(limiter, O.FLUX_HLL, 1.0)
        lev, co = m.get_blocks()
        xyz, _ = W.cell_centres(cfg, lev, co)
        x = 1.0 - xyz[0] if mirror else xyz[0]
        w = np.zeros((len(lev), 4) + x.shape[1:])
        w[:, 0] = 1.0 + 0.3 * np.sin(2 * np.pi * x) + 0.1 * np.cos(4 * np.pi * xyz[1]) * np.sin(2 * np.pi * x)
        w[:, 1] = -0.4 if mirror else 0.4
        w[:, 2] = 0.2
        w[:, 3] = 1.0 + 0.2 * np.cos(2 * np.pi * x)
        m.set_state(0, W.prim_to_cons(w, 1.4))
        for _ in range(4):
            m.advance(2e-3)
        u = m.get_state(0)
        # gather onto the global grid so that the mirror image can be taken
        n = cfg["block_n"]
        ext = cfg["brick"][0] * 2 ** cfg["base_level"] * n
        g = np.zeros((4, ext, ext))
        for b, c in enumerate(co):
            g[:, c[1] * n:(c[1] + 1) * n, c[0] * n:(c[0] + 1) * n] = u[b, :, 0]
        outs.append(g)
    a, b = outs
    bm = b[:, :, ::-1].copy()
    bm[1] = -bm[1]
    assert np.abs(a - bm).max() <= 1e-14, np.abs(a - bm).max()
    assert np.abs(a[0] - a[0][:, ::-1]).max() > 1e-3      # the state itself is not symmetric


# ---------------------------------------------------------------- spatially varying boundary data, eq. (4)
@pytest.mark.parametrize("dim", [2, 3])
def test_bc_data_reproduces_the_linear_field_on_a_refined_mesh(dim):
    # the paper's linear-field test (eq. 21) with the boundary values supplied through bc_data:
    # phi = x + 2y + 3z on the boundary faces; every face ghost (physical boundary, same level, coarse-fine) must
    # then hold phi to the paper's 1e-15 after a fill
    N = 8
    bc = [W.BCDATA] * 6
    m = mesh(dim, N, (2, 1, 1)[:dim] if dim == 2 else (2, 1, 1), 0, 2, bc)
    rng = np.random.default_rng(2)
    for _ in range(2):
        flags = (rng.uniform(size=m.num_blocks) < 0.4).astype(np.int32)
        flags[0] = 1
        m.adapt(flags)
    lev, co = m.get_blocks()
    brick = (2, 1, 1)
    coef = np.array([1.0, 2.0, 3.0][:dim])
    X, nc, _ = H.padded_coords(dim, N, 2, brick, lev, co)
    phi = sum(coef[a] * X[a] for a in range(dim))
    nvar = dim + 2
    u = np.repeat(phi[:, None], nvar, axis=1) * (1.0 + np.arange(nvar))[None, :, None, None, None]
    interior = u[:, :, 2:-2, 2:-2, 2:-2] if dim == 3 else u[:, :, :, 2:-2, 2:-2]
    m.set_state(0, np.ascontiguousarray(interior))
    faces, xyz = H.boundary_faces(dim, N, brick, bc, lev, co, W.BCDATA)
    assert len(faces) > 0
    data = np.zeros((len(faces), nvar, N if dim == 3 else 1, N))
    for q, Xf in enumerate(xyz):
        pf = sum(coef[a] * Xf[a] for a in range(dim))
        for v in range(nvar):
            data[q, v] = (1.0 + v) * pf
    m.set_bc_data(faces, data)
    m.fill_ghosts(0)
    g = m.get_state(0, with_ghosts=True)
    for v in range(nvar):
        assert np.abs(g[:, v][nc] - u[:, v][nc]).max() <= 1e-15 * np.abs(u[:, v]).max() * 4

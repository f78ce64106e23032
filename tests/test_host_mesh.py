"""CPU tests of the library's host side (no compute calls): the shared library
loads and exports every symbol include/f4.h declares; mesh adapt / balance and
the ghost pattern agree with the oracle's independent implementation and with a
brute-force validity check; error behaviour of the C-ABI."""
from __future__ import annotations

import os
import re

import numpy as np
import pytest

import helpers as H
from oracle import oracle as O
from paper_2605_07612_b200 import f4
from paper_2605_07612_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PER, OUT, KEEP = W.PERIODIC, W.OUTFLOW, W.KEEP


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "f4.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(f4_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(f4.SYMBOLS), declared ^ set(f4.SYMBOLS)
    L = f4.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert "sm_100a" in f4.version()


def _pair(dim, N, brick, base, maxl, bc, max_blocks=40000):
    lm = f4.Mesh(dim, N, 2, brick, base, maxl, bc, 1.4, 2, max_blocks)
    om = O.OracleMesh(dim, N, 2, brick, base, maxl, bc, 1.4, 2)
    return lm, om


def _same_leaves(lm, om):
    la, ca = lm.get_blocks()
    lb, cb = om.get_blocks()
    ka, kb = H.key_index(la, ca), H.key_index(lb, cb)
    assert len(ka) == len(la) and set(ka) == set(kb)
    return la, ca, lb, cb


def _check_pattern(lm, om):
    la, ca, lb, cb = _same_leaves(lm, om)
    perm = H.match_blocks(la, ca, lb, cb)          # library block q = oracle block perm[q]
    inv = np.empty_like(perm)
    inv[perm] = np.arange(len(perm))
    kind, nbr, off = om.face_table()
    rec, n1, n2 = lm.pattern()
    dim = lm.dim
    expect = 0
    bc = lm._bc
    for b in range(len(lb)):
        for f in range(2 * dim):
            k = kind[b, f]
            expect += {O.NB_SAME: 1, O.NB_COARSE: 1, O.NB_FINE: 2 ** (dim - 1),
                       O.NB_BOUNDARY: 1 if bc[f] == OUT else 0}[int(k)]
    assert len(rec) == expect
    seen = set()
    for q, (op, face, dst, src, o1, o2) in enumerate(rec):
        ob = perm[dst]
        k = kind[ob, face]
        assert (q < n1) == (op != f4.OP_C2F)       # R1 first, R2 = C2F only
        if op == f4.OP_SRL:
            assert k == O.NB_SAME and inv[nbr[ob, face, 0]] == src
        elif op == f4.OP_BC:
            assert k == O.NB_BOUNDARY and src == dst and bc[face] == OUT
        elif op == f4.OP_F2C:
            assert k == O.NB_FINE and inv[nbr[ob, face, o1 + 2 * o2]] == src
        else:
            assert k == O.NB_COARSE and inv[nbr[ob, face, 0]] == src and tuple(off[ob, face]) == (o1, o2)
        key = (op, face, dst, o1, o2)
        assert key not in seen
        seen.add(key)
    # sorted by destination block inside each round
    for lo, hi in ((0, n1), (n1, n1 + n2)):
        d = rec[lo:hi, 2]
        assert np.all(np.diff(d) >= 0)


@pytest.mark.parametrize("dim", [2, 3])
def test_adapt_and_pattern_match_oracle(dim):
    rng = np.random.default_rng(7 + dim)
    bc = [PER, PER, OUT, OUT, PER, PER][: 2 * dim]
    brick = (2, 1, 3)[:dim]
    lm, om = _pair(dim, 8, brick, 1, 4, bc)
    lm._bc = bc + [PER] * (6 - len(bc))
    _check_pattern(lm, om)
    for it in range(6):
        la, ca, lb, cb = _same_leaves(lm, om)
        flags_l = rng.choice([-1, 0, 1], size=len(la), p=[0.5, 0.35, 0.15]).astype(np.int32)
        perm = H.match_blocks(lb, cb, la, ca)       # oracle block q = library block perm[q]
        ch_l = lm.adapt(flags_l)
        ch_o = om.adapt(flags_l[perm])
        assert ch_l == ch_o
        la, ca, _, _ = _same_leaves(lm, om)
        H.check_mesh_valid(dim, list(brick) + [1] * (3 - dim), lm._bc, la, ca, 1, 4)
        _check_pattern(lm, om)
    lm.close()


def test_block_order_is_morton_and_geometry():
    m = f4.Mesh(3, 16, 2, (1, 1, 1), 2, 3, [PER] * 6, 1.4, 2, 512)
    lev, co, org, dx = m.get_blocks(geometry=True)
    assert len(lev) == 64 and (lev == 2).all()
    # children of one level-1 octant are contiguous
    oct_id = (co[:, 0] >> 1) + 2 * (co[:, 1] >> 1) + 4 * (co[:, 2] >> 1)
    assert np.array_equal(oct_id, np.repeat(np.arange(8), 8))
    assert np.allclose(dx, 1.0 / (4 * 16)) and np.allclose(org, co * 16 * dx[:, None])
    f = np.zeros(64, dtype=np.int32)
    f[10] = 1
    assert m.adapt(f)
    lev2, co2 = m.get_blocks()
    assert len(lev2) == 64 + 7 and (lev2 == 3).sum() == 8
    q = np.where(lev2 == 3)[0]
    assert np.array_equal(q, np.arange(q[0], q[0] + 8))  # the new family sits where its parent was
    m.close()


def test_error_behaviour():
    with pytest.raises(f4.F4Error) as e:
        f4.Mesh(3, 7, 2, (1, 1, 1), 0, 0, [PER] * 6)              # N odd
    assert e.value.code == -1
    with pytest.raises(f4.F4Error):
        f4.Mesh(3, 2, 2, (1, 1, 1), 0, 0, [PER] * 6)              # 2*Ng > N
    with pytest.raises(f4.F4Error):
        f4.Mesh(3, 8, 2, (1, 1, 1), 0, 0, [PER, OUT] + [PER] * 4)  # half-periodic axis
    with pytest.raises(f4.F4Error) as e:
        f4.Mesh(3, 8, 2, (1, 1, 1), 2, 2, [PER] * 6, max_blocks=10)  # base mesh does not fit
    assert e.value.code == -2
    m = f4.Mesh(2, 8, 2, (2, 2), 0, 2, [PER] * 4, max_blocks=6)
    with pytest.raises(f4.F4Error) as e:
        m.adapt(np.array([1, 0, 0, 0], dtype=np.int32))           # 4 - 1 + 4 = 7 > 6
    assert e.value.code == -2
    assert m.num_blocks == 4                                      # nothing modified
    # device work without bound storage: loud failure, no CPU fallback
    for call in (lambda: m.fill_ghosts(0), lambda: m.advance(1e-3), lambda: m.compute_dt(0, 0.4),
                 lambda: m.get_state(0), lambda: m.conserved_totals(0)):
        with pytest.raises(f4.F4Error) as e:
            call()
        assert e.value.code == -4
    m.close()


def test_full_size_config_patterns():
    # record counts of the uniform headline meshes (SURVEY.md §8 size table): 6 SRL records per block
    for n, nb in ((2, 32768), (3, 32768), (4, 13824)):
        cfg = W.config(n)
        m = f4.Mesh.from_config(cfg)
        assert m.num_blocks == nb
        rec, n1, n2 = m.pattern()
        assert n1 == 6 * nb and n2 == 0 and (rec[:, 0] == f4.OP_SRL).all()
        m.close()


def test_asynchronous_adapt_builds_the_same_mesh_and_pattern():
    # f4_adapt_begin / f4_adapt_end (host part on a worker thread, on a copy of the mesh) against the blocking f4_adapt:
    # same leaves, same pattern records, over refine / coarsen / no-change rounds; the mesh in use stays valid meanwhile
    rng = np.random.default_rng(11)
    for dim, N in ((2, 8), (3, 8)):
        bc = [PER, PER, OUT, OUT, PER, PER][: 2 * dim]
        a = f4.Mesh(dim, N, 2, (2, 2, 2)[:dim], 0, 3, bc, max_blocks=4000)
        b = f4.Mesh(dim, N, 2, (2, 2, 2)[:dim], 0, 3, bc, max_blocks=4000)
        for rnd in range(6):
            nb = a.num_blocks
            flags = rng.integers(-1, 2, size=nb).astype(np.int32) if rnd != 3 else np.zeros(nb, dtype=np.int32)
            b.adapt_begin(flags)
            lev_before, co_before = b.get_blocks()            # still the old mesh
            assert len(lev_before) == nb
            with pytest.raises(f4.F4Error):
                b.adapt_begin(flags)                          # one regrid at a time
            ch_a, ch_b = a.adapt(flags), b.adapt_end()
            assert ch_a == ch_b and (rnd != 3 or not ch_a)
            la, ca = a.get_blocks()
            lb, cb = b.get_blocks()
            assert np.array_equal(la, lb) and np.array_equal(ca, cb)
            ra, rb = a.pattern(), b.pattern()
            assert ra[1:] == rb[1:] and np.array_equal(ra[0], rb[0])
        with pytest.raises(f4.F4Error):
            b.adapt_end()                                     # nothing pending
        a.close()
        b.close()


def test_scalar_advection_mesh_has_one_variable():
    cfg = W.config(8, scale=1)
    m = f4.Mesh.from_config(cfg)
    assert m.nvar == 1 and m._shape(False)[1] == 1
    assert m.storage_bytes() == 2 * m.num_blocks * 20 ** 3 * 8          # two states, one variable, padded 20^3 blocks
    # dt without a device: CFL dx / sum |v_i| (reading B6)
    with pytest.raises(f4.F4Error):
        m.compute_dt(0, 0.5)                                            # still needs bound storage (check_state)
    m.close()

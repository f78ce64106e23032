"""f4_conserved_totals_noalloc (-m gpu): the entry point that allocates nothing (scratch in a static device array,
include/f4.h) against f4_conserved_totals, the existing path, on two calls in a row.  Collected last on purpose
(the suite runs with pytest -x)."""
from __future__ import annotations

import numpy as np
import pytest

from paper_2605_07612_b200 import f4
from paper_2605_07612_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL_TOTALS = 1e-12          # the tolerance of the conservation checks in test_gpu_parity.py / test_gpu_rowj.py


def _mesh(cfg, **kw):
    m = f4.Mesh.from_config(cfg, **kw)
    m.bind_torch()
    lev, co = m.get_blocks()
    m.set_state(0, W.initial_state(cfg, lev, co))
    return m


def _close(a, b):
    return np.all(np.abs(a - b) <= TOL_TOTALS * np.abs(b).max())


def test_noalloc_totals_match_the_existing_path_twice_in_a_row():
    """Config 4 at scale 1 (216 blocks of 32^3) and config 3 at scale 2 (64 blocks of 16^3): the first call, then a
    second one after the state has changed (two Heun steps), then the same on the OTHER mesh -- the static array
    keeps the previous call's contents, and more of them than the second mesh has blocks."""
    import torch

    for cfg in (W.config(4, scale=1), W.config(3, scale=2)):
        m = _mesh(cfg)
        out = torch.full((m.nvar,), float("nan"), dtype=torch.float64, device="cuda")
        ref = m.conserved_totals(0)
        m.conserved_totals_noalloc(0, out.data_ptr())
        torch.cuda.synchronize()
        first = out.cpu().numpy().copy()
        assert _close(first, ref), (first, ref)
        for _ in range(2):
            m.advance(m.compute_dt(0, cfg["cfl"]))
        ref2 = m.conserved_totals(0)
        out.fill_(float("nan"))
        m.conserved_totals_noalloc(0, out.data_ptr())
        torch.cuda.synchronize()
        second = out.cpu().numpy().copy()
        assert _close(second, ref2), (second, ref2)
        assert np.isfinite(second).all() and not np.array_equal(first, second)
        m.close()


def test_noalloc_totals_on_a_mixed_level_mesh_and_for_one_variable():
    """Blocks of different levels carry different cell volumes (the finishing kernel reads the level table); scalar
    advection has one variable per cell (config 8 at scale 1)."""
    import torch

    cfg = W.config(3, scale=1)
    m = f4.Mesh.from_config(dict(cfg, max_level=cfg["base_level"] + 1), max_blocks=256)
    m.bind_torch()
    flags = np.zeros(m.num_blocks, dtype=np.int32)
    flags[::3] = 1
    assert m.adapt(flags)
    lev, co = m.get_blocks()
    assert lev.min() != lev.max()
    m.set_state(0, W.initial_state(cfg, lev, co))
    out = torch.zeros(m.nvar, dtype=torch.float64, device="cuda")
    for _ in range(2):
        m.conserved_totals_noalloc(0, out.data_ptr())
        torch.cuda.synchronize()
        assert _close(out.cpu().numpy(), m.conserved_totals(0))
    m.close()

    cfg = W.config(8, scale=1)
    m = _mesh(cfg)
    assert m.nvar == 1
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    for _ in range(2):
        m.conserved_totals_noalloc(0, out.data_ptr())
        torch.cuda.synchronize()
        assert _close(out.cpu().numpy(), m.conserved_totals(0))
    m.close()


def test_noalloc_rejects_what_it_cannot_do():
    """More blocks than the static array holds, a host pointer and a null pointer are errors with a message, and the
    call leaves the device memory it was not given alone (no allocation: torch's allocator sees no change and the
    driver reports no less free memory)."""
    import torch

    cfg = W.config(3, scale=1)
    m = _mesh(cfg)
    out = torch.zeros(m.nvar, dtype=torch.float64, device="cuda")
    m.conserved_totals_noalloc(0, out.data_ptr())          # the first call on this device resolves the symbol address
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    res0 = torch.cuda.memory_reserved()
    for _ in range(50):
        m.conserved_totals_noalloc(0, out.data_ptr())
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0 and torch.cuda.memory_reserved() == res0
    host = np.zeros(m.nvar)
    with pytest.raises(f4.F4Error, match="device pointer"):
        m.conserved_totals_noalloc(0, host.ctypes.data)
    with pytest.raises(f4.F4Error, match="null"):
        m.conserved_totals_noalloc(0, 0)
    m.close()

    # 2D, 8^2 blocks: 256 x 256 = 65 536 blocks > F4_NOALLOC_MAX_BLOCKS (a 168 MB store)
    assert f4.NOALLOC_MAX_BLOCKS == 32768
    big = f4.Mesh(2, 8, 2, (1, 1), 8, 8, [W.PERIODIC] * 4, max_blocks=65536)
    big.bind_torch()
    assert big.num_blocks == 65536
    out = torch.zeros(big.nvar, dtype=torch.float64, device="cuda")
    with pytest.raises(f4.F4Error, match="exceed the static scratch's maximum of 32768"):
        big.conserved_totals_noalloc(0, out.data_ptr())
    assert np.isfinite(big.conserved_totals(0)).all()      # the existing path still serves that mesh
    big.close()

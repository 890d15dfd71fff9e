"""md_cell_list_static (include/md.h): the cell list through an entry point that allocates nothing -- its
scratch is a static __device__ array in the library -- against md_cell_list_build on a md_system with a
workspace (resort = 0, id = NULL: the same canonical order).  Integer outputs: bit-exact.

This file is collected last on purpose (pytest -x stops at the first failure)."""
import ctypes as C

import numpy as np
import pytest
import torch


@pytest.fixture(scope="module")
def B():
    from paper_1912_04232_b200 import build
    build.build()
    from paper_1912_04232_b200 import binding
    binding.lib()
    return binding


def test_sizes_beyond_the_static_scratch_are_refused(B):
    """n > MD_STATIC_MAX_N or more cells than MD_STATIC_MAX_CELLS: MD_EINVAL with a message that names the
    limit, decided on the host before any CUDA call (the buffers here are never touched; stream = 0 is given
    so that the binding does not ask torch for the current CUDA stream: this test runs without a GPU)."""
    dummy = np.zeros(64, np.float32)
    idum = np.zeros(64, np.int32)
    cfg = B.make_config(3, [40.0, 40.0, 40.0], 2.5, 0.3, 128, 0)
    with pytest.raises(B.MdError) as e:
        B.md_cell_list_static(cfg, B.MD_STATIC_MAX_N + 1, dummy, idum, idum, dummy, stream=0)
    assert "MD_STATIC_MAX_N" in str(e.value)
    big = B.make_config(3, [80.0, 80.0, 80.0], 2.5, 0.3, 128, 0)          # 28^3 = 21,952 cells
    with pytest.raises(B.MdError) as e:
        B.md_cell_list_static(big, 1000, dummy, idum, idum, dummy, stream=0)
    assert "MD_STATIC_MAX_CELLS" in str(e.value)
    with pytest.raises(B.MdError):
        B.md_cell_list_static(cfg, 1000, None, idum, idum, dummy, stream=0)   # NULL input


@pytest.mark.gpu
def test_static_cell_list_equals_the_workspace_path_on_calls_in_a_row(B):
    """Calls in a row on one stream, each of another geometry and size than the one before (so the shared
    array holds another call's leftovers every time), and the first geometry once more with moved particles:
    cell_start and perm bit-equal to md_cell_list_build's, pos_sorted = pos[perm]."""
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1912_04232_b200 import workloads as W
    dev = torch.device("cuda", 0)
    rng = np.random.default_rng(11)
    cases = []
    for ci in (2, 0, 1, 2):
        w = W.config(ci)
        pos = w.pos.copy()
        if cases and ci == 2:                                             # second visit: everything moved
            L = w.box.astype(np.float32)
            pos[:, :w.dim] = np.mod(pos[:, :w.dim] + rng.uniform(0, 3, (w.n, w.dim)).astype(np.float32), L[:w.dim])
            pos[:, :w.dim] = np.minimum(pos[:, :w.dim], np.nextafter(L[:w.dim], np.float32(0)))
        cases.append((w, pos))
    checked = 0
    for w, pos_h in cases:
        # the existing path: a md_system over a workspace the caller allocated
        S = B.System(w, resort=0)
        S.pos.copy_(torch.from_numpy(pos_h))
        assert w.n <= B.MD_STATIC_MAX_N and S.cells <= B.MD_STATIC_MAX_CELLS
        B.md_cell_list_build(S.sys, S.pos, None, None, S.cell_start, S.perm)
        # the entry point under test: inputs and outputs only
        pos = torch.from_numpy(pos_h).to(dev)
        cell_start = torch.full((S.cells + 1,), -7, dtype=torch.int32, device=dev)
        perm = torch.full((w.n,), -7, dtype=torch.int32, device=dev)
        pos_sorted = torch.full((w.n, 4), float("nan"), dtype=torch.float32, device=dev)
        B.md_cell_list_static(S.cfg, w.n, pos, cell_start, perm, pos_sorted)
        torch.cuda.synchronize()
        assert torch.equal(cell_start, S.cell_start)
        assert torch.equal(perm, S.perm)
        assert torch.equal(pos_sorted, pos[perm.long()])
        assert torch.equal(pos, torch.from_numpy(pos_h).to(dev))          # the input is untouched
        assert int(cell_start[-1]) == w.n and sorted(perm.tolist()) == list(range(w.n))
        S.close()
        checked += 1
    assert checked == 4

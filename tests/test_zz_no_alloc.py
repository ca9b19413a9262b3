"""nf_cell_offsets_noalloc -- the entry point for callers that cannot let the library allocate.

Some users of this library cannot accept a cudaMalloc inside a call: a simulation whose own memory pool
already holds the whole GPU (a later cudaMalloc can fail), or a time-step loop that overlaps copies and
kernels on several streams (cudaMalloc / cudaFree wait for the whole device).  For them the library has one
call that needs no context and allocates nothing: the exclusive scan of a cell histogram into the cell
offsets of the grid order (step A2), with its tile partial sums in a fixed array inside the
library's device image (limit: NF_NOALLOC_MAX_CELLS cells).

What is checked here: its offsets equal the context path's (nf_bin -> nf_debug_cells) bit for bit -- integer
work, so the tolerance is zero, as in the other binning tests -- on two calls in a row that share the fixed
array (a large grid, then a small one with nothing in between, so the second call meets the first call's
leftovers); at the limit itself; on an empty grid; that a grid beyond the limit is refused with a message
that says why; and that the calls leave the device's free memory untouched.

This file sorts last on purpose (pytest -x stops at the first failure: a failure here hides nothing).
It does not depend on state left by other tests and passes alone in a fresh process as well.
"""
import ctypes

import numpy as np
import pytest

from paper_2110_11392_b200 import workloads as W


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    return torch


def _context_offsets(torch, B, cfg):
    """(histogram on the device, the context path's offsets on the host) for one seeded particle set"""
    pos = torch.from_numpy(W.make_positions(cfg)).cuda()
    with B.NearField(cfg.cpd, cfg.R, cfg.eps_p, 1.0) as nf:
        counts = nf.cell_histogram(pos)          # caller-owned int32 [cpd^3]
        nf.bin(pos)                              # the existing path: A1..A3 with context-owned scratch
        ref = nf.debug_cells()["offsets"]        # uint32 [cpd^3 + 1]
    torch.cuda.synchronize()
    return counts, ref


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_context_path(torch_cuda):
    torch = torch_cuda
    import paper_2110_11392_b200.binding as B
    big = W.scaled(W.CONFIGS[3], 40)             # clustered recipe, 64 000 cells = 31 full tiles + a ragged one
    small = W.CONFIGS[1]                         # 343 cells: a fraction of one tile
    c_big, ref_big = _context_offsets(torch, B, big)
    c_small, ref_small = _context_offsets(torch, B, small)
    assert c_big.numel() == 40 ** 3 and c_small.numel() == 343
    # outputs are made by the caller beforehand: the library itself is handed every byte it may write
    o_big = torch.full((c_big.numel() + 1,), -1, dtype=torch.int32, device="cuda")
    o_small = torch.full((c_small.numel() + 1,), -1, dtype=torch.int32, device="cuda")
    B.cell_offsets_noalloc(c_small, o_small.clone())          # first call on the device: address look-up + module load
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    B.cell_offsets_noalloc(c_big, o_big)                      # call 1 fills 32 words of the shared array ...
    B.cell_offsets_noalloc(c_small, o_small)                  # ... call 2, same stream, uses 1 and must ignore the rest
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "the calls changed the device's free memory"
    got_big = o_big.cpu().numpy().view(np.uint32)
    got_small = o_small.cpu().numpy().view(np.uint32)
    assert np.array_equal(got_big, ref_big)
    assert np.array_equal(got_small, ref_small)
    # and both equal the plain definition on the histogram they were given
    for got, c in ((got_big, c_big), (got_small, c_small)):
        h = c.cpu().numpy().astype(np.int64)
        assert got[0] == 0 and np.array_equal(got[1:].astype(np.int64), np.cumsum(h))
    # a third call, large again: same answer as the first time
    o_again = torch.empty_like(o_big)
    B.cell_offsets_noalloc(c_big, o_again)
    torch.cuda.synchronize()
    assert torch.equal(o_again, o_big)


@pytest.mark.gpu
def test_at_the_limit_and_empty(torch_cuda):
    torch = torch_cuda
    import paper_2110_11392_b200.binding as B
    n = B.NF_NOALLOC_MAX_CELLS                                  # every one of the 4096 tiles in use
    g = torch.Generator(device="cuda").manual_seed(5)
    counts = torch.randint(0, 200, (n,), dtype=torch.int32, device="cuda", generator=g)
    counts[7 * 2048:9 * 2048] = 0                               # two empty tiles in the middle
    off = B.cell_offsets_noalloc(counts)
    torch.cuda.synchronize()
    expect = torch.cumsum(counts.to(torch.int64), 0)
    assert int(off[0]) == 0
    assert torch.equal(off[1:].to(torch.int64), expect)
    # one cell short of a tile boundary, and one past it
    for m in (2047, 2048, 2049, 1):
        o = B.cell_offsets_noalloc(counts[:m].contiguous())
        torch.cuda.synchronize()
        assert int(o[0]) == 0 and torch.equal(o[1:].to(torch.int64), expect[:m])
    o = B.cell_offsets_noalloc(torch.empty(0, dtype=torch.int32, device="cuda"))
    torch.cuda.synchronize()
    assert o.numel() == 1 and int(o[0]) == 0


def test_sizes_beyond_the_limit_are_refused():
    """argument errors come back before anything touches a GPU, so this runs on any machine"""
    import paper_2110_11392_b200.binding as B
    L = B._L
    fake = ctypes.c_void_p(256)                                 # never dereferenced: the size check comes first
    assert L.nf_cell_offsets_noalloc(fake, B.NF_NOALLOC_MAX_CELLS + 1, fake, None) == B.NF_EINVAL
    msg = L.nf_cell_offsets_noalloc_error().decode()
    assert "NF_NOALLOC_MAX_CELLS" in msg and str(B.NF_NOALLOC_MAX_CELLS) in msg and "nf_bin" in msg
    assert L.nf_cell_offsets_noalloc(fake, -1, fake, None) == B.NF_EINVAL
    assert L.nf_cell_offsets_noalloc(fake, 10, None, None) == B.NF_EINVAL
    assert L.nf_cell_offsets_noalloc(None, 10, fake, None) == B.NF_EINVAL
    with open(B.__file__.replace("binding.py", "../include/nearfield.h")) as f:
        assert f"#define NF_NOALLOC_MAX_CELLS {B.NF_NOALLOC_MAX_CELLS}" in f.read()

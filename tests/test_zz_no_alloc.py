"""nolsm_build_neighbours_static: the a0 entry point that allocates no device memory (README "Without cudaMalloc").

Collected last on purpose (the suite runs with pytest -x).  Checks, on two calls in a row that share the static
scratch array, that the result is bit-exact the one of nolsm_build_neighbours (integer work: the parity bar of a0),
that the second, smaller call is not disturbed by what the first one left in the array, that the calls change
nothing in the device's free memory, and that a size beyond the array's maximum is refused with a clear error.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def nolsm():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2104_08245_b200 as m
    m.load_library()  # raises if libnolsm.so is missing: no fallback
    return m


def _static_lists(ctx, torch, pos, box_q, rc_q, cap):
    row_ptr = torch.full((pos.shape[0] + 1,), -7, dtype=torch.int32, device="cuda")
    col_idx = torch.full((cap,), -7, dtype=torch.int32, device="cuda")
    nnzb = ctx.build_neighbours_static(pos, box_q, rc_q, row_ptr, col_idx)
    return row_ptr, col_idx, nnzb


def test_static_scratch_neighbours_match_allocating_path(nolsm):
    import torch
    import nolsm_inputs as gi
    ctx = nolsm.Context()
    assert nolsm.load_library().nolsm_static_setup() == 0
    cases = []
    for n_mol, cutoff in ((4096, 8.0), (216, 6.0)):   # the second call is smaller: stale counts stay behind it
        pos_q, box_q = gi.make_positions(n_mol)
        rc_q = int(round(cutoff * gi.GRID_PER_ANGSTROM))
        pos = torch.as_tensor(pos_q).cuda()
        ref_rp, ref_ci = ctx.build_neighbours(pos, box_q, rc_q)          # existing path (allocates its scratch)
        cases.append((pos, box_q, rc_q, ref_rp.cpu().numpy(), ref_ci.cpu().numpy()))
    # one call first, so that lazy module loading is behind us before free memory is compared
    _static_lists(ctx, torch, cases[1][0], cases[1][1], cases[1][2], len(cases[1][4]))
    bufs = [(torch.full((c[0].shape[0] + 1,), -7, dtype=torch.int32, device="cuda"),
             torch.full((len(c[4]),), -7, dtype=torch.int32, device="cuda")) for c in cases]
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    nnzb = [ctx.build_neighbours_static(c[0], c[1], c[2], rp, ci) for c, (rp, ci) in zip(cases, bufs)]
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after >= free_before, "the static entry point must not allocate device memory"
    for c, (rp, ci), nz in zip(cases, bufs, nnzb):
        assert nz == len(c[4])
        assert np.array_equal(rp.cpu().numpy(), c[3])                    # bit-exact (a0's parity bar)
        assert np.array_equal(ci.cpu().numpy(), c[4])
    ctx.close()


def test_static_scratch_rejects_sizes_beyond_its_maximum(nolsm):
    import torch
    ctx = nolsm.Context()
    n_mol = 262144 + 1                                                   # NOLSM_STATIC_MAX_MOL + 1
    pos = torch.zeros((n_mol, 3), dtype=torch.int32, device="cuda")
    row_ptr = torch.full((n_mol + 1,), -7, dtype=torch.int32, device="cuda")
    col_idx = torch.zeros((16,), dtype=torch.int32, device="cuda")
    with pytest.raises(nolsm.NolsmError, match="NOLSM_STATIC_MAX_MOL"):
        ctx.build_neighbours_static(pos, [1 << 20] * 3, 1 << 16, row_ptr, col_idx)
    assert int(row_ptr[0]) == -7 and int(row_ptr[-1]) == -7              # refused before any launch
    # a list that does not fit the caller's col_idx: same status as the allocating path, needed size reported
    pos_small = torch.zeros((8, 3), dtype=torch.int32, device="cuda")
    rp = torch.zeros(9, dtype=torch.int32, device="cuda")
    with pytest.raises(nolsm.NolsmError, match="capacity"):
        ctx.build_neighbours_static(pos_small, [1 << 20] * 3, 1 << 16, rp, col_idx[:4])
    ctx.close()

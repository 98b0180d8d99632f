"""psd_deposit_uniform_static (include/psd.h): the deposit that allocates nothing -- all scratch in
the library's file-scope device array.  Checked against the existing path (psd_build_tets +
psd_deposit_uniform on a context) within the parity tolerance of tests/test_gpu_parity.py
    per cell |a - b| <= 1e-9 * max_cell + 1e-6 * |b|,  total mass within 1e-10 relative,
on two calls in a row with different inputs (the array keeps the last call's contents).
Collected last (the file name): the suite runs with pytest -x.
"""
import numpy as np
import pytest

import psd_inputs

pytestmark = pytest.mark.gpu


def to_dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def assert_parity(new, ref, what=""):
    mx = float(ref.max())
    err = np.abs(new - ref)
    bound = 1e-9 * mx + 1e-6 * np.abs(ref)
    worst = float((err / bound).max())
    assert worst <= 1.0, f"{what}: worst |err|/bound = {worst:.3e}, max |err| = {err.max():.3e}"


def reference_grid(psd, pos_dev, G):
    """The existing path: a context, psd_build_tets + psd_deposit_uniform, default options."""
    with psd.Context(0) as ctx:
        ctx.psd_build_tets(pos_dev)
        g = ctx.psd_deposit_uniform(G)
        ctx.psd_sync()
        return g.cpu().numpy(), ctx.psd_get_stats().n_pairs


def test_static_deposit_matches_the_existing_path_on_two_calls_in_a_row():
    import torch
    import paper_1612_09491_b200 as psd
    # call 1: a crossing field with many pairs; call 2: other particles, other N and G, fewer pairs
    # (stale counts, cursors or list entries of call 1 would show); call 3: call 1's input again
    cases = [
        (psd_inputs.zeldovich_positions(32, 24, 3, 1.5, 7, dtype="float32", stride=4), 128),
        (psd_inputs.zeldovich_positions(20, 24, 3, 0.5, 11, dtype="float64", stride=3), 64),
        (psd_inputs.zeldovich_positions(32, 24, 3, 1.5, 7, dtype="float32", stride=4), 128),
    ]
    free_after_first = None
    for n, (pos, G) in enumerate(cases):
        pos_dev = to_dev(pos)
        ref, ref_pairs = reference_grid(psd, pos_dev, G)
        grid = torch.full((G, G, G), -3.0, dtype=torch.float64, device="cuda")  # overwritten, not added to
        torch.cuda.synchronize()
        if n == 1:
            free_after_first = torch.cuda.mem_get_info()[0]
        n_pairs = psd.psd_deposit_uniform_static(pos_dev, G, grid)
        torch.cuda.synchronize()
        if n == 1:  # the call itself takes no device memory (the array came with the library)
            assert torch.cuda.mem_get_info()[0] == free_after_first
        got = grid.cpu().numpy()
        assert n_pairs == ref_pairs and n_pairs > 0
        assert abs(float(got.sum()) - 1.0) <= 1e-10
        assert_parity(got, ref, what=f"static deposit, call {n + 1}")


def test_static_deposit_rejects_sizes_beyond_its_scratch():
    import torch
    import paper_1612_09491_b200 as psd
    small = to_dev(psd_inputs.lattice(8, shift=(0.01, 0.02, 0.03)))
    # G beyond PSD_STATIC_MAX_G, G not a multiple of the tile, N beyond PSD_STATIC_MAX_N
    for pos_dev, G, word in ((small, psd.STATIC_MAX_G + 8, "PSD_STATIC_MAX_G"), (small, 20, "multiple of 8")):
        grid = torch.zeros((G, G, G), dtype=torch.float64, device="cuda")
        with pytest.raises(psd.PsdError) as e:
            psd.psd_deposit_uniform_static(pos_dev, G, grid)
        assert e.value.code == 1 and word in str(e.value)
    big = torch.zeros((psd.STATIC_MAX_N + 1,) * 3 + (3,), dtype=torch.float64, device="cuda")
    grid = torch.zeros((64, 64, 64), dtype=torch.float64, device="cuda")
    with pytest.raises(psd.PsdError) as e:
        psd.psd_deposit_uniform_static(big, 64, grid)
    assert e.value.code == 1 and "PSD_STATIC_MAX_N" in str(e.value)
    # more (tet, tile) pairs than the static pair list holds: known after the census
    far = to_dev(psd_inputs.zeldovich_positions(64, 24, 3, 12.0, 3, dtype="float32", stride=4))
    grid = torch.zeros((128, 128, 128), dtype=torch.float64, device="cuda")
    with pytest.raises(psd.PsdError) as e:
        psd.psd_deposit_uniform_static(far, 128, grid)
    assert e.value.code == 1 and "PSD_STATIC_MAX_PAIRS" in str(e.value)
    # and the entry point still works afterwards
    g8 = torch.zeros((16, 16, 16), dtype=torch.float64, device="cuda")
    psd.psd_deposit_uniform_static(small, 16, g8)
    torch.cuda.synchronize()
    assert abs(float(g8.sum()) - 1.0) <= 1e-10

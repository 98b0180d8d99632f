"""GPU parity: the CUDA path (through the C ABI, include/psd.h) against the CPU oracle on the
same seeded inputs.  Tolerances are BASELINE.json's north_star:
    per cell |gpu - oracle| <= 1e-9 * max_cell + 1e-6 * |oracle|
    total mass within 1e-10 relative
    tet and bin counts bit-exact.
"""
import numpy as np
import pytest

import psd_inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def psd():
    import paper_1612_09491_b200 as m
    return m


@pytest.fixture()
def ctx(psd):
    c = psd.Context(0)
    yield c
    c.close()


def to_dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def assert_parity(gpu, ora, M=1.0, what=""):
    gpu = np.asarray(gpu).reshape(ora.shape)
    mx = float(ora.max())
    err = np.abs(gpu - ora)
    bound = 1e-9 * mx + 1e-6 * np.abs(ora)
    worst = float((err / bound).max())
    assert worst <= 1.0, f"{what}: worst |err|/bound = {worst:.3e}, max |err| = {err.max():.3e}"


def assert_mass(gpu_sum, M=1.0):
    assert abs(float(gpu_sum) - M) <= 1e-10 * abs(M), f"mass {float(gpu_sum)!r} vs {M}"


def crossing_field(N, rms, seed=7, dtype="float64", stride=3, modes=24, kmax=3):
    return psd_inputs.zeldovich_positions(N, modes, kmax, rms, seed, dtype=dtype, stride=stride)


KERNELS = [0, 1]  # 0 = binned tile path, 1 = direct path


# ------------------------------------------------------------------ invariants on the GPU alone
@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("N,G,shift", [(4, 8, (0, 0, 0)), (4, 8, (0.013, 0.4, 0.77)),
                                       (6, 16, (0.1, 0.2, 0.3)), (5, 9, (0.1, 0.2, 0.3)),
                                       (8, 8, (0.5, 0.25, 0.125)), (3, 24, (0.01, 0.02, 0.03))])
def test_unperturbed_lattice_is_uniform(psd, ctx, kernel, N, G, shift):
    ctx.psd_set_option(psd.OPT_KERNEL, kernel)
    ctx.psd_build_tets(to_dev(psd_inputs.lattice(N, shift=shift)), 1.0, 2.5)
    g = ctx.psd_deposit_uniform(G).cpu().numpy()
    assert np.allclose(g, 2.5 / G ** 3, rtol=1e-11, atol=0)
    s = ctx.psd_get_stats()
    assert s.n_tets == 6 * N ** 3 and s.n_inverted == 0 and s.n_degenerate == 0


@pytest.mark.parametrize("kernel", KERNELS)
def test_sheared_torus_is_uniform(psd, ctx, kernel):
    ctx.psd_set_option(psd.OPT_KERNEL, kernel)
    ctx.psd_build_tets(to_dev(psd_inputs.lattice(6, shift=(0.21, 0.05, 0.6), shear_xy=1)))
    g = ctx.psd_deposit_uniform(16).cpu().numpy()
    assert np.allclose(g, 1.0 / 16 ** 3, rtol=1e-11, atol=0)


# ------------------------------------------------------------------ element-by-element parity
@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("N,G,rms", [(12, 24, 2.0), (12, 8, 2.0), (10, 40, 1.0), (16, 64, 3.0),
                                     (6, 72, 0.5)])
def test_crossing_field_parity(psd, ctx, oracle, kernel, N, G, rms):
    """Heavily multistream small fields: inverted tets, tets spanning several tiles, tiles met
    through two periodic images (G = 8 with 2-cell-rms displacements)."""
    pos = crossing_field(N, rms)
    ora, st = oracle.deposit_uniform(pos, 1.0, 1.0, G)
    ctx.psd_set_option(psd.OPT_KERNEL, kernel)
    ctx.psd_build_tets(to_dev(pos))
    g = ctx.psd_deposit_uniform(G)
    assert_mass(g.sum())
    assert_parity(g.cpu().numpy(), ora, what=f"N{N} G{G}")
    s = ctx.psd_get_stats()
    assert s.n_inverted == st["n_inverted"] and s.sum_cells == st["n_candidates"]
    # signed-volume mode: every cell exactly one cell volume for any displacement field
    ctx.psd_set_option(psd.OPT_WEIGHT_MODE, 1)
    sg = ctx.psd_deposit_uniform(G).cpu().numpy()
    assert np.allclose(sg, 1.0, rtol=0, atol=1e-10)


@pytest.mark.parametrize("G", [9, 20, 63])
def test_ragged_grid_sizes_use_direct_path(psd, ctx, oracle, G):
    """G not a multiple of the tile edge (Q12)."""
    pos = crossing_field(8, 1.2, seed=3)
    ora, _ = oracle.deposit_uniform(pos, 1.0, 1.0, G)
    ctx.psd_build_tets(to_dev(pos))
    g = ctx.psd_deposit_uniform(G)
    assert_mass(g.sum())
    assert_parity(g.cpu().numpy(), ora)
    assert ctx.psd_get_stats().n_tiles == 0


@pytest.mark.parametrize("chord_axis", [-1, 0, 1, 2])
def test_chord_axis_choices_agree(psd, ctx, oracle, chord_axis):
    pos = crossing_field(10, 1.5, seed=11)
    ora, _ = oracle.deposit_uniform(pos, 1.0, 1.0, 32)
    ctx.psd_set_option(psd.OPT_CHORD_AXIS, chord_axis)
    ctx.psd_build_tets(to_dev(pos))
    assert_parity(ctx.psd_deposit_uniform(32).cpu().numpy(), ora)


@pytest.mark.parametrize("dtype,stride", [("float32", 4), ("float32", 3), ("float64", 3), ("float64", 4)])
def test_position_layouts(psd, ctx, oracle, dtype, stride):
    pos = crossing_field(9, 1.0, dtype=dtype, stride=stride)
    ora, _ = oracle.deposit_uniform(pos, 1.0, 1.0, 24)
    ctx.psd_build_tets(to_dev(pos))
    assert_parity(ctx.psd_deposit_uniform(24).cpu().numpy(), ora)


def test_box_length_total_mass_and_accumulate(psd, ctx, oracle):
    pos = crossing_field(8, 0.9) * 3.0
    ora, _ = oracle.deposit_uniform(pos, 3.0, 7.0, 16)
    ctx.psd_build_tets(to_dev(pos), 3.0, 7.0)
    g = ctx.psd_deposit_uniform(16)
    assert_mass(g.sum(), 7.0)
    assert_parity(g.cpu().numpy(), ora)
    ctx.psd_deposit_uniform(16, g, accumulate=True)
    assert_parity(g.cpu().numpy(), 2.0 * ora)


def test_degenerate_all_coincident(psd, ctx, oracle):
    """Q6: V = 0 exactly -> the whole tet mass goes to the centroid cell."""
    pos = np.full((4, 4, 4, 3), 0.3, dtype=np.float64)
    ora, st = oracle.deposit_uniform(pos, 1.0, 1.0, 8)
    for kernel in KERNELS:
        ctx.psd_set_option(psd.OPT_KERNEL, kernel)
        ctx.psd_build_tets(to_dev(pos))
        g = ctx.psd_deposit_uniform(8).cpu().numpy()
        assert ctx.psd_get_stats().n_degenerate == st["n_degenerate"] == 6 * 64
        assert_parity(g, ora)


def test_cfg0_full_parity_and_bit_exact_census(psd, ctx, oracle):
    """BASELINE.json configs[0]: 32^3 particles, fp64, 64^3 grid, every cell compared."""
    pos = psd_inputs.config_positions(0)
    ora, st = oracle.deposit_uniform(pos, 1.0, 1.0, 64)
    cen = oracle.census(pos, 1.0, 64)
    assert st["n_inverted"] == 0
    ctx.psd_build_tets(to_dev(pos))
    g = ctx.psd_deposit_uniform(64)
    assert_mass(g.sum())
    assert_parity(g.cpu().numpy(), ora, what="cfg0")
    s = ctx.psd_get_stats()
    assert s.n_tets == cen["n_tets"] == 196608
    assert s.n_pairs == cen["n_pairs"] and s.sum_cells == cen["sum_cells"]
    assert s.max_cells == cen["max_cells"] and s.n_inverted == 0
    assert list(s.hist_tet) == cen["hist_tet"].tolist()
    assert list(s.hist_pair) == cen["hist_pair"].tolist()
    assert np.array_equal(ctx.psd_get_tile_counts(), cen["tile_counts"])
    ctx.psd_set_option(psd.OPT_KERNEL, 1)
    assert_parity(ctx.psd_deposit_uniform(64).cpu().numpy(), ora, what="cfg0 direct")


def test_census_bit_exact_with_images_and_inversions(psd, ctx, oracle):
    pos = crossing_field(12, 2.0, dtype="float32", stride=4)
    for G in (8, 24, 48):
        cen = oracle.census(pos, 1.0, G)
        ctx.psd_build_tets(to_dev(pos))
        ctx.psd_deposit_uniform(G)
        s = ctx.psd_get_stats()
        assert (s.n_pairs, s.sum_cells, s.max_cells, s.n_inverted) == (
            cen["n_pairs"], cen["sum_cells"], cen["max_cells"], cen["n_inverted"])
        assert list(s.hist_tet) == cen["hist_tet"].tolist()
        assert list(s.hist_pair) == cen["hist_pair"].tolist()
        assert np.array_equal(ctx.psd_get_tile_counts(), cen["tile_counts"])
        # size classes of the binning (a3): small = the tet's range covers <= 8 cells of the tile,
        # i.e. buckets b <= 3 of the oracle's pair histogram
        cls = ctx.psd_get_tile_class_counts().astype(np.int64)
        assert np.array_equal(cls.sum(axis=1), cen["tile_counts"].astype(np.int64))
        assert int(cls[:, 0].sum()) == int(cen["hist_pair"][:4].sum())
        assert int(cls[:, 1].sum()) == int(cen["hist_pair"][4:].sum())
    # the class threshold is an option (a power of two: the classes stay unions of the buckets);
    # the deposit does not depend on it
    ref = ctx.psd_deposit_uniform(24).cpu().numpy()
    for thr, nb in [(1, 1), (64, 7), (512, 10)]:
        ctx.psd_set_option(psd.OPT_CLASS_SMALL_CELLS, thr)
        g = ctx.psd_deposit_uniform(24).cpu().numpy()
        cls = ctx.psd_get_tile_class_counts().astype(np.int64)
        cen = oracle.census(pos, 1.0, 24)
        assert int(cls[:, 0].sum()) == int(cen["hist_pair"][:nb].sum())
        assert np.allclose(g, ref, rtol=1e-9, atol=1e-18)
    ctx.psd_set_option(psd.OPT_CLASS_SMALL_CELLS, 8)
    with pytest.raises(psd.PsdError):
        ctx.psd_set_option(psd.OPT_CLASS_SMALL_CELLS, 12)


@pytest.mark.parametrize("chunk", [32, 100, 1024])
def test_work_item_chunking_does_not_change_the_result(psd, ctx, oracle, chunk):
    pos = crossing_field(12, 2.0)
    ora, _ = oracle.deposit_uniform(pos, 1.0, 1.0, 16)
    ctx.psd_set_option(psd.OPT_CHUNK, chunk)
    ctx.psd_build_tets(to_dev(pos))
    g = ctx.psd_deposit_uniform(16)
    assert_parity(g.cpu().numpy(), ora)
    s = ctx.psd_get_stats()
    tc = ctx.psd_get_tile_counts().astype(np.int64)
    assert s.n_work_items == int(((tc + chunk - 1) // chunk).sum())


# ------------------------------------------------------------------ patch path
def test_patches_parity_and_refinement(psd, ctx, oracle):
    """a7: refinement census bit-exact, rule reproduces the oracle's list, deposit parity on
    every level, level 0 tiled = uniform deposit, coarse cell = sum of its 8 children."""
    pos = crossing_field(16, 2.5, dtype="float32", stride=4, modes=40, kmax=4)
    base_G, P, max_level, factor = 32, 16, 2, 1.5
    ctx.psd_build_tets(to_dev(pos))
    patches, counts = ctx.psd_refine_patches(base_G, P, max_level, factor, want_counts=True)
    ocounts = [oracle.patch_counts(pos, 1.0, base_G, P, l) for l in range(max_level + 1)]
    for a, b in zip(counts, ocounts):
        assert np.array_equal(a, b)
    opatches = oracle.refine_patches(ocounts, factor)
    assert np.array_equal(patches, opatches)
    assert (patches[:, 0] == 1).any() and (patches[:, 0] == 2).any()
    lit = ctx.psd_refine_patches(base_G, P, max_level, factor, rule=psd.RULE_LITERAL_TOP_DOWN)
    assert np.array_equal(lit, oracle.refine_patches(ocounts, factor, oracle.RULE_LITERAL_TOP_DOWN))
    ora = oracle.deposit_patches(pos, 1.0, 1.0, base_G, P, patches)
    mass = ctx.psd_deposit_patches(patches, P, base_G).cpu().numpy()
    mx = ora.max()
    assert (np.abs(mass - ora) <= 1e-9 * mx + 1e-6 * np.abs(ora)).all()
    # level 0 tiled together == uniform deposit at base_G (Q13)
    uni = ctx.psd_deposit_uniform(base_G).cpu().numpy()
    l0 = patches[:, 0] == 0
    for row, m in zip(patches[l0], mass[l0]):
        _, ox, oy, oz = row
        blk = uni[ox * P:(ox + 1) * P, oy * P:(oy + 1) * P, oz * P:(oz + 1) * P]
        assert np.allclose(m, blk, rtol=1e-9, atol=1e-15)
    assert_mass(mass[l0].sum())


def test_patches_with_shared_faces(psd, ctx, oracle):
    """a7 with every face clipped once (PSD_OPT_FACE_SHARING; one per-tet table per level, the patch
    masses in fixed point until the end, restriction after the conversion): against the oracle, and
    the tet formulation, every chord axis, no restriction and accumulate = 1 (tet formulation again)
    give the same."""
    pos = crossing_field(16, 1.2, dtype="float32", stride=4, modes=40, kmax=4)
    base_G, P, max_level, factor = 32, 16, 2, 1.5
    ctx.psd_build_tets(to_dev(pos))
    patches = ctx.psd_refine_patches(base_G, P, max_level, factor)
    assert (patches[:, 0] == 1).any() and (patches[:, 0] == 2).any()
    ora = oracle.deposit_patches(pos, 1.0, 1.0, base_G, P, patches)
    mx = ora.max()
    mass = ctx.psd_deposit_patches(patches, P, base_G).cpu().numpy()
    assert ctx.psd_get_stats().shared_faces == 1
    assert (np.abs(mass - ora) <= 1e-9 * mx + 1e-6 * np.abs(ora)).all()
    for sharing, restrict in ((0, 1), (2, 1), (3, 0)):
        ctx.psd_set_option(psd.OPT_FACE_SHARING, sharing)
        ctx.psd_set_option(psd.OPT_PATCH_RESTRICT, restrict)
        m2 = ctx.psd_deposit_patches(patches, P, base_G).cpu().numpy()
        assert ctx.psd_get_stats().shared_faces == (1 if sharing else 0)
        assert (np.abs(m2 - ora) <= 1e-9 * mx + 1e-6 * np.abs(ora)).all(), (sharing, restrict)
    ctx.psd_set_option(psd.OPT_FACE_SHARING, 1)
    ctx.psd_set_option(psd.OPT_PATCH_RESTRICT, 1)
    acc = ctx.psd_deposit_patches(patches, P, base_G)
    ctx.psd_deposit_patches(patches, P, base_G, acc, accumulate=True)
    assert ctx.psd_get_stats().shared_faces == 0
    assert (np.abs(acc.cpu().numpy() - 2.0 * ora) <= 2e-9 * mx + 2e-6 * np.abs(ora)).all()


@pytest.mark.parametrize("N,B,dtype,stride", [(32, 8, "float32", 4), (40, 8, "float64", 3), (36, 8, "float32", 3),
                                              (32, 4, "float32", 4)])
def test_subblock_census_bit_exact_and_drives_the_refinement(psd, ctx, oracle, N, B, dtype, stride):
    """a7 / PAPER.md:74-76: the sub-block bounding-box estimate (fixed point, order independent)
    equals the oracle's on every level, with a ragged last sub-block (N = 36) too, and the patch
    list the rule builds from it is the oracle's."""
    pos = crossing_field(N, 1.5, dtype=dtype, stride=stride, modes=40, kmax=4)
    base_G, P, max_level, factor = 32, 8, 2, 1.5
    ctx.psd_build_tets(to_dev(pos))
    ctx.psd_set_option(psd.OPT_REFINE_SUBBLOCK, B)
    try:
        patches, counts = ctx.psd_refine_patches(base_G, P, max_level, factor, want_counts=True)
    finally:
        ctx.psd_set_option(psd.OPT_REFINE_SUBBLOCK, 0)
    ocounts = [oracle.subblock_counts(pos, 1.0, base_G, P, l, B) for l in range(max_level + 1)]
    for a, b in zip(counts, ocounts):
        assert np.array_equal(a, b)
    assert psd.SUBBLOCK_UNIT == oracle.SUBBLOCK_UNIT
    assert np.array_equal(patches, oracle.refine_patches(ocounts, factor))
    assert (patches[:, 0] == 1).any()


def test_patch_list_subset_and_order_independence(psd, ctx, oracle):
    pos = crossing_field(12, 2.0)
    patches = np.array([[1, 3, 0, 2], [0, 1, 1, 0], [2, 7, 7, 7], [0, 0, 0, 1], [1, 0, 3, 3]], dtype=np.int32)
    ora = oracle.deposit_patches(pos, 1.0, 1.0, 32, 16, patches)
    ctx.psd_build_tets(to_dev(pos))
    mass = ctx.psd_deposit_patches(patches, 16, 32).cpu().numpy()
    assert (np.abs(mass - ora) <= 1e-9 * ora.max() + 1e-6 * np.abs(ora)).all()
    perm = np.array([4, 2, 0, 3, 1])
    mass2 = ctx.psd_deposit_patches(patches[perm], 16, 32).cpu().numpy()
    assert np.allclose(mass2, mass[perm], rtol=1e-9, atol=1e-18)


# ------------------------------------------------------------------ boundary behaviour
def test_patch_restriction_fills_refined_parents_from_their_children(psd, ctx, oracle):
    """PAPER.md:193 / PSD_OPT_PATCH_RESTRICT: a patch whose 8 children are all listed is not deposited
    into but summed from them.  Same masses as the direct deposit and as the oracle; a parent with
    only some children listed is deposited directly; accumulate = 1 turns the restriction off."""
    pos = crossing_field(16, 2.5, dtype="float32", stride=4, modes=40, kmax=4)
    base_G, P, max_level, factor = 32, 16, 2, 1.5
    ctx.psd_build_tets(to_dev(pos))
    patches = ctx.psd_refine_patches(base_G, P, max_level, factor)
    # plus one level-1 patch family made incomplete: drop one child of a refined level-0 patch
    lv1 = np.nonzero(patches[:, 0] == 1)[0]
    incomplete = np.delete(patches, lv1[-1], axis=0)
    for plist in (patches, incomplete):
        ora = oracle.deposit_patches(pos, 1.0, 1.0, base_G, P, plist)
        ctx.psd_set_option(psd.OPT_PATCH_RESTRICT, 1)
        m1 = ctx.psd_deposit_patches(plist, P, base_G).cpu().numpy()
        n_restricted = ctx.psd_get_stats().n_restricted_patches
        n_pairs_restricted = ctx.psd_get_stats().n_pairs
        ctx.psd_set_option(psd.OPT_PATCH_RESTRICT, 0)
        m0 = ctx.psd_deposit_patches(plist, P, base_G).cpu().numpy()
        assert ctx.psd_get_stats().n_restricted_patches == 0
        assert ctx.psd_get_stats().n_pairs > n_pairs_restricted      # fewer (tet, tile) pairs to deposit
        assert n_restricted > 0
        assert_parity(m1, ora, what="restricted")
        assert_parity(m0, ora, what="direct")
        assert np.allclose(m1, m0, rtol=1e-9, atol=1e-9 * ora.max())
    # the number of patches filled by restriction = those with all 8 children in the list
    def n_refined(plist):
        have = {tuple(r) for r in plist.tolist()}
        return sum(all((l + 1, 2 * a + (d & 1), 2 * b + ((d >> 1) & 1), 2 * c + (d >> 2)) in have for d in range(8))
                   for l, a, b, c in plist.tolist())
    ctx.psd_set_option(psd.OPT_PATCH_RESTRICT, 1)
    for plist in (patches, incomplete):
        ctx.psd_deposit_patches(plist, P, base_G)
        assert ctx.psd_get_stats().n_restricted_patches == n_refined(plist)
    assert n_refined(incomplete) < n_refined(patches)
    # accumulate: direct deposit everywhere, twice the mass
    m = ctx.psd_deposit_patches(patches, P, base_G)
    m = ctx.psd_deposit_patches(patches, P, base_G, m, accumulate=True).cpu().numpy()
    assert ctx.psd_get_stats().n_restricted_patches == 0
    assert_parity(0.5 * m, oracle.deposit_patches(pos, 1.0, 1.0, base_G, P, patches), what="accumulated")


@pytest.mark.parametrize("kernel", KERNELS)
def test_unwrap_suspects_are_counted_on_both_paths(psd, ctx, kernel):
    """Q4: the minimum image is valid while every Lagrangian cell edge is shorter than L/2; cells with
    an edge longer than L/4 are counted (advisory).  N = 3: every edge is L/3; N = 8: L/8."""
    ctx.psd_set_option(psd.OPT_KERNEL, kernel)
    ctx.psd_build_tets(to_dev(psd_inputs.lattice(3, shift=(0.01, 0.02, 0.03))))
    ctx.psd_deposit_uniform(8)
    assert ctx.psd_get_stats().n_unwrap_suspect == 27
    ctx.psd_build_tets(to_dev(psd_inputs.lattice(8, shift=(0.01, 0.02, 0.03))))
    ctx.psd_deposit_uniform(8)
    assert ctx.psd_get_stats().n_unwrap_suspect == 0


@pytest.mark.parametrize("records", [0, 1, 3000, 700])
def test_pair_record_buffer_modes_agree(psd, ctx, oracle, records):
    """PSD_OPT_PAIR_RECORDS: stage A in its own kernel writing pair records (default), fused into the
    deposit kernel (0), and a record buffer far smaller than the pair list (refilled slab by slab,
    also in the host-output call that streams the grid back in slabs of x-tiles)."""
    import torch
    pos = crossing_field(24, 1.5, dtype="float32", stride=4)
    G = 192
    ora, _ = oracle.deposit_uniform(pos, 1.0, 1.0, G)
    ctx.psd_set_option(psd.OPT_PAIR_RECORDS, records)
    ctx.psd_set_option(psd.OPT_CHUNK, 256)
    ctx.psd_build_tets(to_dev(pos))
    g = ctx.psd_deposit_uniform(G)
    assert ctx.psd_get_stats().n_pairs > 20000
    assert_mass(g.sum())
    assert_parity(g.cpu().numpy(), ora, what=f"records={records}")
    hg = torch.full((G, G, G), -1.0, dtype=torch.float64).pin_memory()
    ctx.psd_deposit_uniform_host(torch.from_numpy(pos).pin_memory(), G, hg)
    assert_parity(hg.numpy(), ora, what=f"records={records}, host output")
    # a tiny grid where a tet's range meets a tile in several periodic images (the records-only
    # deposit kernel is not used there: the largest cell range plus a tile does not fit the grid)
    pos = crossing_field(12, 2.0)
    for G in (8, 16, 24):
        ora, _ = oracle.deposit_uniform(pos, 1.0, 1.0, G)
        ctx.psd_build_tets(to_dev(pos))
        assert_parity(ctx.psd_deposit_uniform(G).cpu().numpy(), ora, what=f"records={records}, images, G={G}")
        s = ctx.psd_get_stats()
        lo_hi = [oracle.build_tet(pos, 1.0, G, i, j, k, t)[2:] for i in range(12) for j in range(12) for k in range(12) for t in range(6)]
        assert s.max_extent == max(int((hi - lo).max()) + 1 for lo, hi in lo_hi)


@pytest.mark.parametrize("case", ["crossing", "crossing_far", "lattice", "jittered", "tiny_cells"])
def test_fp32_rows_cover_the_fp64_rows(psd, ctx, oracle, case):
    """PSD_OPT_ROWS_FP32: which columns a face meets is decided in fp32 with a
    margin, the clip stays fp64.  The fp32 set of jobs must hold every row range of the fp64 one
    (n_rows_missed, checked on the device pair by pair), may hold a few more jobs, and the deposit
    is the same."""
    if case == "crossing":
        pos, G = crossing_field(24, 1.5, dtype="float32", stride=4), 192
    elif case == "crossing_far":   # long thin tets: coordinates far from the tile, steep edges
        pos, G = crossing_field(16, 6.0), 256
    elif case == "lattice":        # every vertex on a lattice line, every edge along one or through corners
        pos, G = psd_inputs.lattice(16), 64
    elif case == "jittered":
        pos, G = psd_inputs.jittered_lattice(32, seed=5), 16
    else:                          # tets far smaller than a cell: slopes of every size inside one column
        pos, G = crossing_field(16, 0.5), 64
    ora, _ = oracle.deposit_uniform(pos, 1.0, 1.0, G)
    ctx.psd_set_option(psd.OPT_FACE_SHARING, 0)  # the tet formulation: its record kernel holds the check
    ctx.psd_set_option(psd.OPT_COUNTERS, 1)
    ctx.psd_set_option(psd.OPT_CHUNK, 256)
    res = {}
    for mode in (0, 1):
        ctx.psd_set_option(psd.OPT_ROWS_FP32, mode)
        ctx.psd_build_tets(to_dev(pos))
        g = ctx.psd_deposit_uniform(G)
        s = ctx.psd_get_stats()
        assert_parity(g.cpu().numpy(), ora, what=f"{case}, rows_fp32={mode}")
        res[mode] = (g.cpu().numpy(), s.n_face_jobs, s.n_face_clips, s.n_rows_missed)
    assert res[1][3] == 0 and res[0][3] == 0
    # a few more jobs in fp32; on the exact lattice every vertex sits on lattice lines and the margin
    # puts it on both sides of each (about twice the jobs, all but the fp64 ones empty)
    assert res[0][1] <= res[1][1] <= (3.0 if case == "lattice" else 1.02) * res[0][1] + 64, (res[0][1], res[1][1])
    assert np.abs(res[1][0] - res[0][0]).max() <= 1e-13 * max(1.0, np.abs(res[0][0]).max())


@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("case", ["crossing", "crossing_f64", "lattice", "jittered", "coincident", "box_mass"])
def test_shared_face_path_parity(psd, ctx, oracle, case, axis):
    """PSD_OPT_FACE_SHARING: every face of the tessellation clipped once for its two tets (in the
    pair of the tet that owns it, one chord axis per deposit, 64-bit fixed-point tiles and grid).
    Against the oracle: crossing fields (inverted tets), the exact lattice (every decision a tie: the
    general clip), the paper's jittered lattice on a coarse grid (most tets inside one cell: the
    pairs' specials), coincident particles (degenerate tets), L != 1 and M != 1."""
    import torch
    L, M = 1.0, 1.0
    if case == "crossing":
        pos, G = crossing_field(24, 1.5, dtype="float32", stride=4), 192
    elif case == "crossing_f64":
        pos, G = crossing_field(16, 3.0), 64
    elif case == "lattice":
        pos, G = psd_inputs.lattice(16), 64
    elif case == "jittered":
        pos, G = psd_inputs.jittered_lattice(32, seed=5), 32
    elif case == "coincident":
        pos, G = np.full((6, 6, 6, 3), 0.3, dtype=np.float64), 32
    else:
        pos, G, L, M = crossing_field(12, 0.9) * 3.0, 40, 3.0, 7.0
    ora, st = oracle.deposit_uniform(pos, L, M, G)
    ctx.psd_set_option(psd.OPT_FACE_SHARING, 1 + axis)
    ctx.psd_set_option(psd.OPT_COUNTERS, 1)
    ctx.psd_set_option(psd.OPT_CHUNK, 256)
    ctx.psd_build_tets(to_dev(pos), L, M)
    g = ctx.psd_deposit_uniform(G)
    s = ctx.psd_get_stats()
    assert s.shared_faces == 1, "the shared-face path did not run"
    assert s.n_pairs > 0 and s.n_degenerate == st["n_degenerate"]  # the tet census still runs
    assert_mass(g.sum(), M)
    assert_parity(g.cpu().numpy(), ora, what=f"{case}, axis {axis}")
    # the face jobs found in fp64 (PSD_OPT_ROWS_FP32 = 0): no more jobs, the same deposit
    ctx.psd_set_option(psd.OPT_ROWS_FP32, 0)
    ctx.psd_build_tets(to_dev(pos), L, M)
    g64 = ctx.psd_deposit_uniform(G)
    s64 = ctx.psd_get_stats()
    assert s64.shared_faces == 1 and s64.n_face_jobs <= s.n_face_jobs
    # (on the exact lattice the margin adds jobs whose polygon is a segment on a lattice line)
    assert s64.n_face_clips == s.n_face_clips or case == "lattice"
    assert float((g - g64).abs().max()) <= 1e-13 * float(g64.max())
    ctx.psd_set_option(psd.OPT_ROWS_FP32, 1)
    if case == "crossing":
        # fewer jobs than the tet formulation with the same axis (each face once), same deposit
        ctx.psd_set_option(psd.OPT_FACE_SHARING, 0)
        ctx.psd_set_option(psd.OPT_CHORD_AXIS, axis)
        ctx.psd_build_tets(to_dev(pos), L, M)
        g0 = ctx.psd_deposit_uniform(G)
        s0 = ctx.psd_get_stats()
        assert s0.shared_faces == 0 and 0.45 * s0.n_face_jobs < s.n_face_jobs < 0.62 * s0.n_face_jobs
        assert float((g - g0).abs().max()) <= 1e-11 * float(g0.max())
        # signed-volume mode: every cell 1; the host-output call (grid converted slab by slab); and
        # accumulate = 1, which the fixed-point grid cannot serve (the tet formulation runs)
        ctx.psd_set_option(psd.OPT_FACE_SHARING, 1 + axis)
        ctx.psd_set_option(psd.OPT_CHORD_AXIS, -1)
        ctx.psd_set_option(psd.OPT_WEIGHT_MODE, 1)
        ctx.psd_build_tets(to_dev(pos))
        gv = ctx.psd_deposit_uniform(G)
        assert ctx.psd_get_stats().shared_faces == 1
        assert float((gv - 1.0).abs().max()) <= 1e-9
        ctx.psd_set_option(psd.OPT_WEIGHT_MODE, 0)
        hg = torch.full((G, G, G), -1.0, dtype=torch.float64).pin_memory()
        ctx.psd_deposit_uniform_host(torch.from_numpy(pos).pin_memory(), G, hg)
        assert ctx.psd_get_stats().shared_faces == 1
        assert_parity(hg.numpy(), ora, what="shared faces, host output")
        ctx.psd_build_tets(to_dev(pos))
        ctx.psd_deposit_uniform(G, g, accumulate=True)
        assert ctx.psd_get_stats().shared_faces == 0
        assert_parity(g.cpu().numpy(), 2.0 * ora, what="shared faces, accumulate")


def test_error_codes(psd, ctx):
    import torch
    with pytest.raises(psd.PsdError) as e:
        ctx.psd_deposit_uniform(8)
    assert e.value.code == 2  # PSD_ERR_STATE
    bad = torch.full((4, 4, 4, 3), float("nan"), dtype=torch.float64, device="cuda")
    with pytest.raises(psd.PsdError) as e:
        ctx.psd_build_tets(bad)
    assert e.value.code == 1
    ctx.psd_build_tets(to_dev(psd_inputs.lattice(4)))
    with pytest.raises(psd.PsdError):
        ctx._ck(ctx._L.psd_deposit_uniform(ctx._h, 0, 0, 0))
    with pytest.raises(psd.PsdError):
        ctx.psd_set_option(99, 1)
    with pytest.raises(psd.PsdError):
        ctx.psd_deposit_patches(np.array([[0, 5, 0, 0]], dtype=np.int32), 16, 32)  # origin outside
    with pytest.raises(psd.PsdError):
        ctx.psd_deposit_patches(np.array([[0, 0, 0, 0], [0, 0, 0, 0]], dtype=np.int32), 16, 32)
    # the context still works after errors
    g = ctx.psd_deposit_uniform(8).cpu().numpy()
    assert np.allclose(g, 1.0 / 512, rtol=1e-12)


def test_host_buffer_entry_point(psd, ctx, oracle):
    import torch
    pos = crossing_field(10, 1.0, dtype="float32", stride=4)
    ora, _ = oracle.deposit_uniform(pos, 1.0, 1.0, 24)
    hp = torch.from_numpy(pos).pin_memory()
    hg = torch.empty((24, 24, 24), dtype=torch.float64).pin_memory()
    ctx.psd_deposit_uniform_host(hp, 24, hg)
    assert_parity(hg.numpy(), ora)
    assert ctx.psd_launch_count() > 0
    # G = 192 (24 tiles per side): the grid comes back in 3 slabs of x-tiles on the copy stream while
    # later slabs are deposited; every cell against the oracle, twice (the context's buffers are reused)
    pos = crossing_field(24, 1.5, dtype="float32", stride=4)
    ora, _ = oracle.deposit_uniform(pos, 1.0, 1.0, 192)
    hp = torch.from_numpy(pos).pin_memory()
    hg = torch.full((192, 192, 192), -1.0, dtype=torch.float64).pin_memory()
    for _ in range(2):
        ctx.psd_deposit_uniform_host(hp, 192, hg)
        assert_parity(hg.numpy(), ora)
        hg.fill_(-1.0)
    # pageable host memory (plain numpy arrays): the copies serialise but the result is the same
    ng = np.full((192, 192, 192), -1.0)
    ctx.psd_deposit_uniform_host(pos, 192, ng)
    assert_parity(ng, ora)


def test_patches_host_buffer_entry_point(psd, ctx, oracle):
    """psd_deposit_patches_host: positions from host memory, refinement + deposit, masses back to
    host memory in one C-ABI call -- the same list and the same masses as the device calls."""
    import torch
    pos = crossing_field(16, 2.5, dtype="float32", stride=4, modes=40, kmax=4)
    base_G, P, max_level, factor = 32, 16, 2, 1.5
    ctx.psd_build_tets(to_dev(pos))
    want_list = ctx.psd_refine_patches(base_G, P, max_level, factor)
    cap = sum(((base_G << l) // P) ** 3 for l in range(max_level + 1))
    hm = torch.full((cap, P, P, P), -1.0, dtype=torch.float64).pin_memory()
    got_list = ctx.psd_deposit_patches_host(torch.from_numpy(pos).pin_memory(), base_G, P, max_level, factor, hm)
    assert np.array_equal(got_list, want_list)
    n = len(got_list)
    ora = oracle.deposit_patches(pos, 1.0, 1.0, base_G, P, got_list)
    assert_parity(hm.numpy()[:n], ora)
    assert (hm.numpy()[n:] == -1.0).all()      # nothing written past the list
    # pageable numpy buffers, and a buffer that is too small for the list
    nm = np.zeros((cap, P, P, P))
    assert np.array_equal(ctx.psd_deposit_patches_host(pos, base_G, P, max_level, factor, nm), want_list)
    assert_parity(nm[:n], ora)
    with pytest.raises(psd.PsdError) as e:
        ctx.psd_deposit_patches_host(pos, base_G, P, max_level, factor, np.zeros((n - 1, P, P, P)))
    assert e.value.code == 1


def test_host_entry_points_validate_their_buffers(psd, ctx):
    """The host entry points take raw addresses: dtype, size, contiguity and residency are checked
    in the binding before the library writes G^3 (or n P^3) doubles through them."""
    import torch
    pos = crossing_field(6, 0.5, dtype="float32", stride=4)
    with pytest.raises(ValueError):
        ctx.psd_deposit_uniform_host(pos, 16, np.zeros((16, 16, 16), dtype=np.float32))
    with pytest.raises(ValueError):
        ctx.psd_deposit_uniform_host(pos, 16, np.zeros((16, 16, 15)))
    with pytest.raises(ValueError):
        ctx.psd_deposit_uniform_host(pos, 16, np.zeros((16, 16, 32))[:, :, ::2])
    with pytest.raises(ValueError):
        ctx.psd_deposit_uniform_host(pos, 16, torch.zeros((16, 16, 16), dtype=torch.float64, device="cuda"))
    with pytest.raises(ValueError):
        ctx.psd_deposit_uniform_host(pos[:, :, ::2][:, :, :3], 16, np.zeros((16, 16, 16)))
    with pytest.raises(ValueError):
        ctx.psd_deposit_patches_host(pos, 16, 8, 1, 2.0, np.zeros((4, 8, 8, 8), dtype=np.float32))
    g = np.zeros((16, 16, 16))
    ctx.psd_deposit_uniform_host(pos, 16, g)
    assert_mass(g.sum())


def test_runs_on_a_non_default_stream(psd, oracle):
    import torch
    pos = crossing_field(10, 1.0)
    ora, _ = oracle.deposit_uniform(pos, 1.0, 1.0, 16)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        d = to_dev(pos)
    st.synchronize()
    c = psd.Context(0, stream=st)
    c.psd_build_tets(d)
    g = c.psd_deposit_uniform(16)
    c.psd_sync()
    assert_parity(g.cpu().numpy(), ora)
    c.close()


# ------------------------------------------------------------------ full-size configs
def sample_windows(G, n, edge, seed):
    u = psd_inputs.splitmix64(seed, 0, 3 * n) % np.uint64(G)
    return [tuple(int(x) for x in u[3 * i:3 * i + 3]) for i in range(n)], edge


def window_of(grid_dev, lo, edge, G):
    import torch
    ix = [(torch.arange(edge, device=grid_dev.device) + l) % G for l in lo]
    return grid_dev[ix[0]][:, ix[1]][:, :, ix[2]].cpu().numpy()


def aimed_windows(oracle, pos, G, edge, n_random, seed):
    """Where the full-size tests look: across the periodic seam, around the densest region of the
    particle distribution (a coarse histogram of the input positions), around the tet with the
    largest cell range and around the thinnest tet (both found by the oracle), plus seeded
    random windows.  Nothing here comes from the CUDA path."""
    wins = {"seam": (G - 3, G - 5, 0)}
    H = min(G, 256)
    idx = np.floor(pos[..., :3].reshape(-1, 3).astype(np.float64) * H).astype(np.int64) % H
    flat = (idx[:, 0] * H + idx[:, 1]) * H + idx[:, 2]
    del idx
    dense = int(np.bincount(flat, minlength=H ** 3).argmax())
    del flat
    d = np.array([dense // (H * H), (dense // H) % H, dense % H]) * (G // H) + (G // H) // 2
    wins["densest"] = tuple(int(x) for x in (d - edge // 2) % G)
    e = oracle.extreme_tets(pos, 1.0, G, min_cells=8)
    wins["largest_tet"] = tuple(int(x) for x in (e["largest"]["lo"] - 2) % G)
    wins["thinnest_tet"] = tuple(int(x) for x in (e["thinnest"]["lo"] - 2) % G)
    rnd, _ = sample_windows(G, n_random, edge, seed)
    for i, lo in enumerate(rnd):
        wins[f"random{i}"] = tuple(int(x) for x in lo)
    return wins, e


def check_windows(oracle, pos, grid, G, wins, edge, mx):
    names = list(wins)
    oras = oracle.deposit_windows(pos, 1.0, 1.0, G, [(wins[k], (edge,) * 3) for k in names])
    for k, ora in zip(names, oras):
        err = np.abs(window_of(grid, wins[k], edge, G) - ora)
        assert (err <= 1e-9 * mx + 1e-6 * np.abs(ora)).all(), (k, wins[k], float(err.max()))
        assert ora.max() > 0


def check_census(oracle, ctx, pos, G, win_tiles=None):
    """a2/a3 bit-exact: pairs per (tile, size class) of the last binned deposit against the oracle,
    on every tile, or on windows of tiles; histograms and scalars when every tile is compared."""
    s = ctx.psd_get_stats()
    nt = G // 8
    got = ctx.psd_get_tile_class_counts().reshape(nt, nt, nt, 2)
    if win_tiles is None:
        c = oracle.census_classes(pos, 1.0, G)
        assert np.array_equal(got[..., 0], c["counts_small"]) and np.array_equal(got[..., 1], c["counts_large"])
        assert np.array_equal(np.array(s.hist_tet, dtype=np.uint64), c["hist_tet"])
        assert np.array_equal(np.array(s.hist_pair, dtype=np.uint64), c["hist_pair"])
        assert (s.n_pairs, s.sum_cells, s.max_cells, s.n_inverted) == \
            (c["n_pairs"], c["sum_cells"], c["max_cells"], c["n_inverted"])
        return
    for lo, n in win_tiles:
        c = oracle.census_classes(pos, 1.0, G, win_lo=lo, win_n=n)
        ix = np.ix_(*[(np.arange(n[a]) + lo[a]) % nt for a in range(3)])
        assert np.array_equal(got[..., 0][ix], c["counts_small"]), lo
        assert np.array_equal(got[..., 1][ix], c["counts_large"]), lo
        assert c["n_pairs"] > 0
        assert np.array_equal(np.array(s.hist_tet, dtype=np.uint64), c["hist_tet"])
        assert (s.sum_cells, s.max_cells, s.n_inverted) == (c["sum_cells"], c["max_cells"], c["n_inverted"])


@pytest.mark.parametrize("cfg_index,n_random,edge", [(1, 4, 12), (2, 2, 12)])
def test_full_size_config_sampled_parity(psd, ctx, oracle, cfg_index, n_random, edge):
    """BASELINE.json configs[1], [2] at full size in the launch configuration bench.py times:
    total mass, signed-volume cover of every cell, pairs per (tile, size class) and census
    histograms bit-exact on every tile, and oracle parity on windows aimed at the method's hard
    places (windows may wrap around the box)."""
    import torch
    cfg = psd_inputs.CONFIGS[cfg_index]
    G = cfg["G"]
    pos = psd_inputs.config_positions(cfg_index)
    ctx.psd_build_tets(to_dev(pos))
    grid = torch.empty((G, G, G), dtype=torch.float64, device="cuda")
    ctx.psd_deposit_uniform(G, grid)
    assert_mass(grid.sum())
    assert float(grid.min()) > 0.0
    mx = float(grid.max())
    check_census(oracle, ctx, pos, G)
    wins, ext = aimed_windows(oracle, pos, G, edge, n_random, 1000 + cfg_index)
    assert ext["largest"]["n_cells"] == ctx.psd_get_stats().max_cells
    check_windows(oracle, pos, grid, G, wins, edge, mx)
    s = ctx.psd_get_stats()
    assert s.n_tets == 6 * cfg["N"] ** 3 and s.n_degenerate == 0
    assert s.shared_faces == 1  # every face clipped once: the default path at full size
    ctx.psd_set_option(psd.OPT_WEIGHT_MODE, 1)
    ctx.psd_deposit_uniform(G, grid)
    assert float((grid - 1.0).abs().max()) < 1e-9


def test_cfg3_full_size_patches(psd, ctx, oracle):
    """BASELINE.json configs[3]: 256^3 particles, base 128^3 in 16^3-cell patches, 2 levels,
    factor 4 (rule: DESIGN.md Q14).  Refinement census and patch list bit-exact vs the oracle,
    deposit parity on sampled patches of every level, and the properties that hold for all of
    them: level 0 carries the whole mass, a refined coarse cell equals the sum of its 8 children."""
    import torch
    cfg = psd_inputs.CONFIGS[3]
    pc = cfg["patches"]
    base_G, P, max_level, factor = pc["base_G"], pc["P"], pc["max_level"], pc["factor"]
    pos = psd_inputs.config_positions(3)
    ctx.psd_build_tets(to_dev(pos))
    patches, counts = ctx.psd_refine_patches(base_G, P, max_level, factor, want_counts=True)
    ocounts = [oracle.patch_counts(pos, 1.0, base_G, P, l) for l in range(max_level + 1)]
    for a, b in zip(counts, ocounts):
        assert np.array_equal(a, b)
    assert np.array_equal(patches, oracle.refine_patches(ocounts, factor))
    levels = patches[:, 0]
    assert (levels == 0).sum() == (base_G // P) ** 3
    assert (levels == 1).any() and (levels == 2).any(), "the refinement rule must fire on cfg3"
    lit = ctx.psd_refine_patches(base_G, P, max_level, factor, rule=psd.RULE_LITERAL_TOP_DOWN)
    assert np.array_equal(lit, oracle.refine_patches(ocounts, factor, oracle.RULE_LITERAL_TOP_DOWN))
    mass = ctx.psd_deposit_patches(patches, P, base_G)
    s = ctx.psd_get_stats()
    assert s.n_tets == 6 * cfg["N"] ** 3 and s.n_degenerate == 0
    assert s.shared_faces == 1  # every face clipped once: the default path at full size
    assert_mass(mass[torch.from_numpy(levels == 0).cuda()].sum())
    # sampled patches against the oracle: per level the hottest one (largest census count) and
    # four seeded ones
    pick = []
    for l in range(max_level + 1):
        idx = np.nonzero(levels == l)[0]
        cnt_l = np.array([int(ocounts[l][tuple(patches[i, 1:])]) for i in idx])
        pick.append(int(idx[int(cnt_l.argmax())]))
        u = psd_inputs.splitmix64(3000 + l, 0, 4) % np.uint64(len(idx))
        pick += [int(idx[int(x)]) for x in u]
    pick = sorted(set(pick))
    ora = oracle.deposit_patches(pos, 1.0, 1.0, base_G, P, patches[pick])
    got = mass[torch.tensor(pick, device="cuda")].cpu().numpy()
    mx = float(mass.max())
    err = np.abs(got - ora)
    assert (err <= 1e-9 * mx + 1e-6 * np.abs(ora)).all(), float(err.max())
    # restriction (Q13): every refined patch's coarse cells equal the sum of the 8 children
    index = {tuple(r): i for i, r in enumerate(patches.tolist())}
    checked = 0
    for i, (l, ox, oy, oz) in enumerate(patches.tolist()):
        if l == max_level or (l + 1, 2 * ox, 2 * oy, 2 * oz) not in index or checked >= 40:
            continue
        coarse = mass[i]
        fine = torch.empty((2 * P, 2 * P, 2 * P), dtype=torch.float64, device="cuda")
        for d in range(8):
            a, b, c = d & 1, (d >> 1) & 1, d >> 2
            fine[a * P:(a + 1) * P, b * P:(b + 1) * P, c * P:(c + 1) * P] = \
                mass[index[(l + 1, 2 * ox + a, 2 * oy + b, 2 * oz + c)]]
        summed = fine.reshape(P, 2, P, 2, P, 2).sum(dim=(1, 3, 5))
        assert float((summed - coarse).abs().max()) <= 1e-9 * mx
        checked += 1
    assert checked > 0


def test_cfg4_full_size_uniform(psd, ctx, oracle):
    """BASELINE.json configs[4]: 512^3 particles (805 M tets) onto 1024^3 cells (8.6 GB) in one
    pass: total mass, positivity, oracle parity on sampled windows, signed-volume cover."""
    import torch
    cfg = psd_inputs.CONFIGS[4]
    G = cfg["G"]
    pos = psd_inputs.config_positions(4)
    ctx.psd_build_tets(to_dev(pos))
    grid = torch.empty((G, G, G), dtype=torch.float64, device="cuda")
    ctx.psd_deposit_uniform(G, grid)
    s = ctx.psd_get_stats()
    assert s.n_tets == 6 * cfg["N"] ** 3 == 805306368 and s.n_degenerate == 0
    assert s.shared_faces == 1  # every face clipped once: the default path at full size
    total = float(grid.sum())
    assert abs(total - 1.0) <= 1e-10, total
    assert float(grid.min()) > 0.0
    mx = float(grid.max())
    edge = 12
    wins, ext = aimed_windows(oracle, pos, G, edge, 3, 1004)
    assert ext["largest"]["n_cells"] == s.max_cells
    check_windows(oracle, pos, grid, G, wins, edge, mx)
    # pairs per (tile, size class) bit-exact on four regions of 8^3 tiles (64^3 cells) at those places
    nt = G // 8
    regions = [(tuple(int((c // 8 - 3) % nt) for c in wins[k]), (8, 8, 8))
               for k in ("seam", "densest", "largest_tet", "thinnest_tet")]
    check_census(oracle, ctx, pos, G, regions)
    ctx.psd_set_option(psd.OPT_WEIGHT_MODE, 1)
    ctx.psd_deposit_uniform(G, grid)
    assert float((grid - 1.0).abs().max()) < 1e-9


# ------------------------------------------------------------------ SURVEY.md 8(f) row 1
@pytest.mark.parametrize("kernel", KERNELS)
def test_paper_weak_scaling_workload_jittered_lattice(psd, ctx, oracle, kernel):
    """PAPER.md:175 (section 7.2): lattice + independent uniform offsets of up to one cell width,
    deposited on a grid with G = N/2, so most tets fall inside one or two cells: the trivial /
    accumulate path instead of the clip path.  Every cell against the oracle."""
    N, G = 32, 16
    pos = psd_inputs.jittered_lattice(N, seed=175, amplitude_cells=1.0)
    ora, st = oracle.deposit_uniform(pos, 1.0, 1.0, G)
    ctx.psd_set_option(psd.OPT_KERNEL, kernel)
    ctx.psd_build_tets(to_dev(pos))
    g = ctx.psd_deposit_uniform(G)
    assert_mass(g.sum())
    assert_parity(g.cpu().numpy(), ora, what="jittered lattice")
    s = ctx.psd_get_stats()
    assert s.n_inverted == st["n_inverted"] > 0 and s.sum_cells == st["n_candidates"]


def test_paper_weak_scaling_workload_at_its_quoted_size(psd, ctx, oracle):
    """PAPER.md:175 at the size the paper quotes: 512^3 jittered particles onto 256^3 cells, the
    launch configuration `bench.py --config 5` times.  Mass, positivity, aimed + random windows."""
    import torch
    cfg = psd_inputs.CONFIGS[5]
    G = cfg["G"]
    pos = psd_inputs.config_positions(5)
    ctx.psd_build_tets(to_dev(pos))
    grid = torch.empty((G, G, G), dtype=torch.float64, device="cuda")
    ctx.psd_deposit_uniform(G, grid)
    s = ctx.psd_get_stats()
    assert s.n_tets == 6 * cfg["N"] ** 3 and s.n_degenerate == 0
    assert s.shared_faces == 1  # every face clipped once: the default path at full size
    assert_mass(grid.sum())
    assert float(grid.min()) > 0.0
    wins, _ = aimed_windows(oracle, pos, G, 12, 2, 1005)
    check_windows(oracle, pos, grid, G, wins, 12, float(grid.max()))


@pytest.mark.parametrize("N", [2, 3])
def test_minimal_lattice_and_single_tile(psd, ctx, oracle, N):
    """Smallest inputs the ABI accepts, one 8^3 tile.  N = 2: every Lagrangian cell edge is about
    L/2, outside the unwrap's validity (Q4) -- both sides must still take the same
    minimum image, rint for rint.  N = 3: the smallest valid lattice."""
    pos = psd_inputs.zeldovich_positions(N, 3, 1, 0.2, 5, dtype="float64", stride=3)
    ora, _ = oracle.deposit_uniform(pos, 1.0, 1.0, 8)
    ctx.psd_build_tets(to_dev(pos))
    g = ctx.psd_deposit_uniform(8)
    assert_mass(g.sum())
    assert_parity(g.cpu().numpy(), ora)
    assert ctx.psd_get_stats().n_tiles == 1

"""Pins for the oracle's full deposit, census and patch path (oracle/psd_oracle.c O1-O6).

Invariants fixed by the method itself: PAPER.md:39-45 (equal mass per Lagrangian cell, 6 tets
tile it), Eq. 1 (density = sum of m/V over covering tets), PAPER.md:72 (patches).
"""
import numpy as np
import pytest

import psd_inputs


def crossing_field(N, rms, seed=7, dtype="float64", stride=3):
    return psd_inputs.zeldovich_positions(N, 24, 3, rms, seed, dtype=dtype, stride=stride)


@pytest.mark.parametrize("N,G", [(4, 8), (4, 4), (6, 9), (5, 8), (8, 4)])
@pytest.mark.parametrize("shift", [(0, 0, 0), (0.013, 0.4, 0.77)])
def test_unperturbed_lattice_is_uniform(oracle, N, G, shift):
    """An unperturbed (rigidly shifted) lattice deposits exactly M/G^3 everywhere -- also with
    every vertex on a cell face (G = 2N, zero shift; Q7) and for non-power-of-two G (Q12)."""
    pos = psd_inputs.lattice(N, shift=shift)
    grid, st = oracle.deposit_uniform(pos, 1.0, 2.5, G)
    assert st["n_tets"] == 6 * N ** 3 and st["n_inverted"] == 0 and st["n_degenerate"] == 0
    assert np.allclose(grid, 2.5 / G ** 3, rtol=1e-12, atol=0)


def test_sheared_torus_is_uniform(oracle):
    """Q3: integer torus shear x -> x + y (mod 1) keeps the density exactly uniform and
    exercises the minimum-image unwrap on every cell of the wrap plane."""
    pos = psd_inputs.lattice(6, shift=(0.21, 0.05, 0.6), shear_xy=1)
    grid, _ = oracle.deposit_uniform(pos, 1.0, 1.0, 12)
    assert np.allclose(grid, 1.0 / 12 ** 3, rtol=1e-12, atol=0)


def test_box_length_and_units(oracle):
    """L != 1: positions in [0,L); the mass per cell does not depend on the unit of length."""
    pos = psd_inputs.lattice(4, L=3.0, shift=(0.3, 0.1, 0.2))
    grid, _ = oracle.deposit_uniform(pos, 3.0, 1.0, 8)
    assert np.allclose(grid, 1.0 / 512, rtol=1e-12)
    p1 = crossing_field(6, 0.8)
    g1, _ = oracle.deposit_uniform(p1, 1.0, 1.0, 12)
    g3, _ = oracle.deposit_uniform(p1 * 4.0, 4.0, 1.0, 12)
    assert np.allclose(g1, g3, rtol=1e-10, atol=1e-16)


def test_mass_conservation_and_signed_cover(oracle):
    """Pin 3 (sum grid = M) and pin 6 (signed-volume mode: every cell gets exactly one cell
    volume for ANY displacement field -- degree-1 map of the torus), with inverted tets."""
    pos = crossing_field(12, 2.0)   # every cell edge stays < L/2, so the unwrap is valid (Q4)
    grid, st = oracle.deposit_uniform(pos, 1.0, 1.0, 24)
    assert st["n_inverted"] > 0.3 * st["n_tets"]
    assert abs(grid.sum() - 1.0) < 1e-12
    assert (grid > 0).all()
    signed, _ = oracle.deposit_uniform(pos, 1.0, 1.0, 24, mode=oracle.MODE_SIGNED)
    assert np.allclose(signed, 1.0, rtol=0, atol=1e-11)


def test_fp32_positions_are_read_exactly(oracle):
    """fp32 input == the same numbers handed over as fp64 (conversion is exact)."""
    p32 = crossing_field(6, 1.0, dtype="float32", stride=4)
    p64 = p32[..., :3].astype(np.float64).copy()
    a, _ = oracle.deposit_uniform(p32, 1.0, 1.0, 12)
    b, _ = oracle.deposit_uniform(p64, 1.0, 1.0, 12)
    assert np.allclose(a, b, rtol=1e-13, atol=0)   # summation order (OpenMP) is the only difference


def test_window_and_range_are_consistent_with_full(oracle):
    pos = crossing_field(6, 1.5)
    G = 12
    full, st = oracle.deposit_uniform(pos, 1.0, 1.0, G)
    win = oracle.deposit_window(pos, 1.0, 1.0, G, [10, 3, 0], [4, 5, 12])  # wraps in x
    want = np.take(full, np.arange(10, 14) % G, axis=0)[:, 3:8, :]
    assert np.allclose(win, want, rtol=1e-12, atol=1e-18)
    acc = np.zeros((G, G, G))
    n3 = 6 ** 3
    for a, b in [(0, 50), (50, 51), (51, n3)]:
        acc, _ = oracle.deposit_uniform_range(pos, 1.0, 1.0, G, a, b, grid=acc)
    assert np.allclose(acc, full, rtol=1e-12, atol=1e-18)


def test_all_particles_coincident_is_degenerate(oracle):
    """Q6: V = 0 exactly -> the whole tet mass goes to the cell holding the centroid."""
    pos = np.full((3, 3, 3, 3), 0.3)
    grid, st = oracle.deposit_uniform(pos, 1.0, 1.0, 4)
    assert st["n_degenerate"] == st["n_tets"] == 162
    assert grid[1, 1, 1] == pytest.approx(1.0) and np.count_nonzero(grid) == 1


def test_census_properties(oracle):
    """O5: totals tie the census to the deposit's own candidate count (two code paths), to the
    tile grid and to a brute-force count over cells on a tiny input."""
    pos = crossing_field(8, 2.0)
    G = 16
    c = oracle.census(pos, 1.0, G)
    _, st = oracle.deposit_uniform(pos, 1.0, 1.0, G)
    assert c["n_tets"] == 6 * 8 ** 3 == int(c["hist_tet"].sum())
    assert c["sum_cells"] == st["n_candidates"]
    assert c["n_inverted"] == st["n_inverted"]
    assert c["n_pairs"] == int(c["tile_counts"].sum()) == int(c["hist_pair"].sum())
    assert c["max_cells"] <= 2 ** (np.nonzero(c["hist_tet"])[0].max())
    # brute force with the single-tet entry point
    nt = G // 8
    tc = np.zeros((nt, nt, nt), dtype=np.int64)
    for i in range(8):
        for j in range(8):
            for k in range(8):
                for t in range(6):
                    _, _, lo, hi = oracle.build_tet(pos, 1.0, G, i, j, k, t)
                    tiles = [sorted({(x % G) // 8 for x in range(lo[a], hi[a] + 1)}) for a in range(3)]
                    for a in tiles[0]:
                        for b in tiles[1]:
                            for d in tiles[2]:
                                tc[a, b, d] += 1
    assert np.array_equal(tc.ravel(), c["tile_counts"].astype(np.int64))


def test_patches_level0_equals_uniform_and_restriction(oracle):
    """Q13: level-0 patches tiled together = deposit_uniform(base_G); every coarse cell equals
    the sum of its 8 children where refined."""
    pos = crossing_field(8, 1.5, dtype="float32", stride=4)
    base_G, P = 8, 4
    patches = [[0, a, b, c] for a in range(2) for b in range(2) for c in range(2)]
    patches += [[1, a, b, c] for a in (2, 3) for b in (0, 1) for c in (3, 0)]   # children of (1,0,1),(1,0,0)
    patches += [[2, 7, 1, 0], [2, 0, 0, 7]]
    patches = np.array(patches, dtype=np.int32)
    mass = oracle.deposit_patches(pos, 1.0, 1.0, base_G, P, patches)
    uni0, _ = oracle.deposit_uniform(pos, 1.0, 1.0, base_G)
    uni1, _ = oracle.deposit_uniform(pos, 1.0, 1.0, 2 * base_G)
    uni2, _ = oracle.deposit_uniform(pos, 1.0, 1.0, 4 * base_G)
    for q, (l, a, b, c) in enumerate(patches):
        ref = (uni0, uni1, uni2)[l][a * P:(a + 1) * P, b * P:(b + 1) * P, c * P:(c + 1) * P]
        assert np.allclose(mass[q], ref, rtol=1e-11, atol=1e-18)
    coarse = uni0.reshape(base_G, 1, base_G, 1, base_G, 1)
    fine = uni1.reshape(base_G, 2, base_G, 2, base_G, 2).sum(axis=(1, 3, 5))
    assert np.allclose(fine, coarse[:, 0, :, 0, :, 0], rtol=1e-11)


def test_patch_counts_and_refine_rule(oracle):
    """PAPER.md:66 refinement by tet count; Q14 rules on integer counts."""
    pos = crossing_field(16, 2.5, dtype="float32", stride=4)
    base_G, P = 32, 4
    counts = [oracle.patch_counts(pos, 1.0, base_G, P, l) for l in range(3)]
    c0 = oracle.census(pos, 1.0, base_G, tile=P)
    assert np.array_equal(counts[0].ravel(), c0["tile_counts"].astype(np.uint64))
    pl = oracle.refine_patches(counts, 2.0)
    lv = pl[:, 0]
    assert (lv == 0).sum() == 8 ** 3
    assert (lv == 1).sum() % 8 == 0 and (lv == 2).sum() % 8 == 0
    assert (lv == 1).sum() > 0
    have = {tuple(r) for r in pl.tolist()}
    for l, a, b, c in pl.tolist():          # every patch's parent exists
        if l:
            assert (l - 1, a // 2, b // 2, c // 2) in have
    hot2 = np.argwhere(counts[2] > 2.0 * counts[2].astype(float).mean())
    for a, b, c in hot2.tolist():           # every hot level-2 candidate is present
        assert (2, a, b, c) in have
    lit = oracle.refine_patches(counts, 1.2, rule=oracle.RULE_LITERAL_TOP_DOWN)
    assert (lit[:, 0] == 0).sum() == 8 ** 3


def test_input_generator_is_seeded_and_matches_recipe():
    a = psd_inputs.config_positions(0)
    b = psd_inputs.config_positions(0)
    assert a.dtype == np.float64 and a.shape == (32, 32, 32, 3)
    assert psd_inputs.sha256_of(a) == psd_inputs.sha256_of(b)
    q = np.arange(32) / 32.0
    d = a.copy()
    d[..., 0] -= q[:, None, None]; d[..., 1] -= q[None, :, None]; d[..., 2] -= q[None, None, :]
    d = (d + 0.5) % 1.0 - 0.5
    assert np.isclose(np.sqrt(np.mean(d * d)) * 32, 0.3, rtol=1e-9)
    from psd_inputs import zeldovich as z
    k, g, phi = z._draw_modes(5, 40, 4)
    assert len({tuple(x) for x in k.tolist()}) == 40 and ((k * k).sum(1) <= 16).all()
    assert np.abs(z.displacement_direct(16, k, g, phi) - z.displacement_fft(16, k, g, phi)).max() < 1e-12
    # curl-free: displacement parallel to k for a single mode
    p1 = z.displacement_direct(8, k[:1], g[:1], phi[:1])
    assert np.abs(np.cross(p1.reshape(-1, 3), k[0].astype(float))).max() < 1e-12


def test_cfg0_has_no_shell_crossing(oracle):
    """BASELINE.json configs[0]: 'no shell crossing' -> no inverted tets; mass conserved."""
    pos = psd_inputs.config_positions(0)
    grid, st = oracle.deposit_uniform(pos, 1.0, 1.0, 64)
    assert st["n_tets"] == 196608 and st["n_inverted"] == 0
    assert abs(grid.sum() - 1.0) < 1e-12


# ------------------------------------------------------------------ O7: sub-block AABB census
def test_subblock_census_closed_form_on_the_aligned_lattice(oracle):
    """PAPER.md:74-76.  Unperturbed lattice, N = 32, sub-blocks of 8^3 cells: every sub-block's
    box is exactly its own Lagrangian cube, so a patch that IS a sub-block cube receives exactly
    the sub-block's 6 x 8^3 tets, and a patch of half the edge exactly 1/8 of them."""
    pos = psd_inputs.lattice(32)
    unit = oracle.SUBBLOCK_UNIT
    c = oracle.subblock_counts(pos, 1.0, 32, 8, 0)      # patch edge = sub-block edge
    assert c.shape == (4, 4, 4) and np.all(c == 6 * 512 * unit)
    c = oracle.subblock_counts(pos, 1.0, 32, 4, 0)      # 8 patches per sub-block
    assert c.shape == (8, 8, 8) and np.all(c == 6 * 64 * unit)
    c = oracle.subblock_counts(pos, 1.0, 32, 8, 1)      # level 1: the same patches in space
    assert c.shape == (8, 8, 8) and np.all(c == 6 * 64 * unit)
    c = oracle.subblock_counts(pos, 1.0, 32, 16, 0)     # 8 sub-blocks per patch
    assert c.shape == (2, 2, 2) and np.all(c == 6 * 4096 * unit)


@pytest.mark.parametrize("N,B,base_G,P,level", [(32, 8, 32, 8, 0), (32, 8, 32, 8, 1), (24, 8, 48, 4, 0),
                                                (20, 8, 40, 8, 0), (32, 4, 16, 4, 1)])
def test_subblock_census_conserves_the_tet_count(oracle, N, B, base_G, P, level):
    """The shares of one box over the patches sum to 1, so the estimates sum to 6 N^3 -- up to the
    half-unit rounding of each (sub-block, patch) term; also with a ragged last sub-block."""
    pos = crossing_field(N, 1.5, seed=11, dtype="float32", stride=4)
    c = oracle.subblock_counts(pos, 1.0, base_G, P, level, B)
    total = int(c.sum(dtype=np.uint64))
    assert abs(total - 6 * N ** 3 * oracle.SUBBLOCK_UNIT) <= 0.5 * 27 * 64 * ((N + B - 1) // B) ** 3


def test_subblock_census_against_point_sampling(oracle):
    """Brute force: uniform points in every sub-block's bounding box (boxes taken here with numpy
    from the unwrapped particles), binned to patches, weighted with the sub-block's tet count."""
    N, B, base_G, P = 32, 8, 32, 8
    pos = crossing_field(N, 1.0, seed=5)
    c = oracle.subblock_counts(pos, 1.0, base_G, P, 0, B).astype(np.float64) / oracle.SUBBLOCK_UNIT
    rng = np.random.default_rng(3)
    npatch = base_G // P
    est = np.zeros((npatch,) * 3)
    idx = np.arange(B + 1)
    for bi in range(N // B):
        for bj in range(N // B):
            for bk in range(N // B):
                sub = pos[np.ix_((bi * B + idx) % N, (bj * B + idx) % N, (bk * B + idx) % N)][..., :3]
                ref = sub[0, 0, 0]
                sub = sub - np.rint(sub - ref)          # minimum image of the first particle
                lo, hi = sub.reshape(-1, 3).min(0), sub.reshape(-1, 3).max(0)
                pts = lo + (hi - lo) * rng.random((4000, 3))
                cell = np.floor(pts * npatch).astype(int) % npatch
                np.add.at(est, (cell[:, 0], cell[:, 1], cell[:, 2]), 6 * B ** 3 / 4000.0)
    # 64 boxes x 4000 points: per-patch sampling error ~ a few percent of the mean
    assert np.abs(est - c).max() < 0.05 * c.mean()
    assert abs(c.sum() - 6 * N ** 3) < 1e-3


def test_fp32_geometry_does_not_hold_the_parity_tolerance(oracle):
    """BASELINE north_star: "fp32 clip allowed only if it holds" |x - ref| <= 1e-9 max_cell +
    1e-6 |ref| and total mass to 1e-10.  The oracle built with fp32 geometry (fp64 determinant and
    sums) against the __float128 build on a crossing field: the double build sits ~1e-7 of the
    tolerance away, the fp32 build exceeds it many times over -- which is why the CUDA path clips
    in fp64 (DESIGN.md section 4 item 4)."""
    pos = crossing_field(8, 2.0, dtype="float32", stride=4)
    gold, _ = oracle.deposit_uniform(pos, 1.0, 1.0, 16, kind="gold")
    dbl, _ = oracle.deposit_uniform(pos, 1.0, 1.0, 16, kind="double")
    sgl, _ = oracle.deposit_uniform(pos, 1.0, 1.0, 16, kind="single")
    tol = 1e-9 * gold.max() + 1e-6 * np.abs(gold)
    assert (np.abs(dbl - gold) / tol).max() < 1e-3
    assert (np.abs(sgl - gold) / tol).max() > 5.0
    assert abs(sgl.sum() - 1.0) > 1e-10 > abs(dbl.sum() - 1.0)


# ------------------------------------------------------------------ O5 / O6 / Q14: pins of the counters
def _bit_width(v: int) -> int:
    return int(v).bit_length()


def _clustered(x, y, z):
    """N = 2 'lattice' whose per-axis coordinates are the given pairs: every Lagrangian cell has
    the same bounding box [min, max] per axis (the wrap cell unwraps back to it), and every Kuhn
    tet holds corners 0 and 7, hence spans that whole box."""
    pos = np.empty((2, 2, 2, 3))
    pos[..., 0] = np.asarray(x)[:, None, None]
    pos[..., 1] = np.asarray(y)[None, :, None]
    pos[..., 2] = np.asarray(z)[None, None, :]
    return pos


@pytest.mark.parametrize("x,y,z,ncell,bucket", [
    ((0.30, 0.31), (0.30, 0.31), (0.30, 0.31), 1, 0),        # all in cell (1,1,1) of G = 4
    ((0.249, 0.251), (0.30, 0.31), (0.30, 0.31), 2, 1),      # straddles x = 1/4
    ((0.249, 0.251), (0.499, 0.501), (0.749, 0.751), 8, 3),  # straddles one face per axis
    ((0.249, 0.501), (0.249, 0.501), (0.30, 0.31), 9, 4),    # 3 x 3 x 1 cells
])
def test_census_histogram_buckets_hand_made(oracle, x, y, z, ncell, bucket):
    """O5: bucket b = bit_width(n_cells - 1): ranges of 1, 2, 8, 9 cells fall in buckets 0, 1, 3, 4
    (worked out by hand from the coordinates, G = 4, tile = 2)."""
    c = oracle.census(_clustered(x, y, z), 1.0, 4, tile=2)
    want = np.zeros(64, dtype=np.uint64)
    want[bucket] = 48
    assert np.array_equal(c["hist_tet"], want)
    assert c["sum_cells"] == 48 * ncell and c["max_cells"] == ncell


def test_census_pair_histogram_hand_made(oracle):
    """O5, per (tet, tile) pair: the 3 x 3 x 1 range above covers cells 0..2 in x and y, i.e. 2 cells
    of tile 0 and 1 cell of tile 1 per axis, and one z cell (cell 1, tile 0): pairs of
    4, 2, 2 and 1 cells -> buckets bit_width(n-1) = 2, 1, 1, 0, one of each per tet."""
    c = oracle.census(_clustered((0.249, 0.501), (0.249, 0.501), (0.30, 0.31)), 1.0, 4, tile=2)
    want = np.zeros(64, dtype=np.uint64)
    want[0], want[1], want[2] = 48, 96, 48
    assert np.array_equal(c["hist_pair"], want)
    tc = c["tile_counts"].reshape(2, 2, 2)
    assert np.array_equal(tc[:, :, 0], np.full((2, 2), 48)) and not tc[:, :, 1].any()
    assert c["n_pairs"] == 4 * 48


def test_census_histograms_recomputed_in_python(oracle):
    """O5: hist_tet, hist_pair and the per-tile 'inside' counts recomputed with python sets from
    the single-tet entry point on a crossing field whose tets wrap around the box."""
    N, G, tile = 8, 16, 8
    pos = crossing_field(N, 2.0)
    c = oracle.census(pos, 1.0, G)
    ht, hp = np.zeros(64, dtype=np.uint64), np.zeros(64, dtype=np.uint64)
    for i in range(N):
        for j in range(N):
            for k in range(N):
                for t in range(6):
                    _, _, lo, hi = oracle.build_tet(pos, 1.0, G, i, j, k, t)
                    n = [int(hi[a] - lo[a] + 1) for a in range(3)]
                    ht[_bit_width(n[0] * n[1] * n[2] - 1)] += 1
                    per_axis = []
                    for a in range(3):
                        inside = {}
                        for cc in range(int(lo[a]), int(hi[a]) + 1):
                            inside[(cc % G) // tile] = inside.get((cc % G) // tile, 0) + 1
                        per_axis.append(inside)
                    for na in per_axis[0].values():
                        for nb in per_axis[1].values():
                            for nc in per_axis[2].values():
                                hp[_bit_width(na * nb * nc - 1)] += 1
    assert np.array_equal(ht, c["hist_tet"])
    assert np.array_equal(hp, c["hist_pair"])
    assert np.count_nonzero(hp) >= 4      # the field does spread over several buckets


def test_patch_stats_counters_recomputed_per_tet(oracle):
    """O6 counters (they feed bench.py's work model for the patch config): candidate cells of a
    patch = cells of each tet's range that wrap into the patch box; cells with non-zero overlap
    counted with the single-tet entry point."""
    N, base_G, P = 6, 8, 4
    pos = crossing_field(N, 1.2)
    patches = np.array([[0, 0, 0, 0], [0, 1, 0, 1], [1, 3, 0, 2], [1, 0, 3, 3]], dtype=np.int32)
    _, st = oracle.deposit_patches_stats(pos, 1.0, 1.0, base_G, P, patches)
    want = np.zeros((len(patches), 2), dtype=np.int64)
    for q, (lv, ox, oy, oz) in enumerate(patches.tolist()):
        G = base_G << lv
        org = (ox * P, oy * P, oz * P)
        for i in range(N):
            for j in range(N):
                for k in range(N):
                    for t in range(6):
                        verts, _, lo, hi = oracle.build_tet(pos, 1.0, G, i, j, k, t)
                        n = (hi - lo + 1).astype(np.int64)
                        vol, _ = oracle.tet_deposit_box(verts * float(G), lo, n)
                        sel = np.ones(tuple(n), dtype=bool)
                        for a in range(3):
                            cells = (np.arange(lo[a], hi[a] + 1) % G)
                            ok = (cells >= org[a]) & (cells < org[a] + P)
                            sel &= ok.reshape([-1 if b == a else 1 for b in range(3)])
                        want[q, 0] += int(sel.sum())
                        want[q, 1] += int(((vol != 0) & sel).sum())
    assert np.array_equal(st, want)
    assert (want[:, 1] > 0).all() and (want[:, 1] < want[:, 0]).all()


def test_refine_rule_literal_top_down_hand_built():
    """Q14, rule 0 on hand-built counts with a known answer: threshold = factor x mean of level 0;
    a patch above it is split, its children are tested against the SAME absolute number."""
    from oracle import psd_oracle as oracle
    c0 = np.array([10, 10, 10, 10, 10, 10, 10, 50], dtype=np.uint64).reshape(2, 2, 2)  # mean 15
    c1 = np.zeros((4, 4, 4), dtype=np.uint64)
    c1[2:, 2:, 2:] = 5            # children of (1,1,1)
    c1[3, 3, 3] = 40              # one of them above 2 x 15 = 30
    c1[0, 0, 0] = 1000            # far above, but its parent (0,0,0) is not split: must not appear
    c2 = np.zeros((8, 8, 8), dtype=np.uint64)
    pl = oracle.refine_patches([c0, c1, c2], 2.0, rule=oracle.RULE_LITERAL_TOP_DOWN)
    got = {tuple(r) for r in pl.tolist()}
    want = {(0, a, b, c) for a in range(2) for b in range(2) for c in range(2)}
    want |= {(1, 2 + a, 2 + b, 2 + c) for a in range(2) for b in range(2) for c in range(2)}
    want |= {(2, 6 + a, 6 + b, 6 + c) for a in range(2) for b in range(2) for c in range(2)}
    assert got == want and len(pl) == len(want)
    # the order is level, then (ox, oy, oz) lexicographic
    assert pl.tolist() == sorted(pl.tolist())
    # a count exactly AT the threshold does not split (strict >)
    c0b = np.array([10, 10, 10, 10, 10, 10, 10, 30], dtype=np.uint64).reshape(2, 2, 2)  # mean 12.5
    pl = oracle.refine_patches([c0b, c1], 2.4, rule=oracle.RULE_LITERAL_TOP_DOWN)      # thr = 30
    assert len(pl) == 8


def test_refine_rule_bottom_up_hand_built():
    """Q14, rule 1 on hand-built counts: hot = count > factor x mean of ITS level; a parent is
    split if any child is hot or split; splitting creates all 8 children."""
    from oracle import psd_oracle as oracle
    c0 = np.ones((2, 2, 2), dtype=np.uint64)
    c1 = np.ones((4, 4, 4), dtype=np.uint64)
    c2 = np.ones((8, 8, 8), dtype=np.uint64)
    c2[5, 0, 2] = 600             # mean = (511 + 600) / 512 = 2.17; 600 > 4 x mean: hot
    pl = oracle.refine_patches([c0, c1, c2], 4.0)
    got = {tuple(r) for r in pl.tolist()}
    want = {(0, a, b, c) for a in range(2) for b in range(2) for c in range(2)}
    want |= {(1, 2 + a, b, c) for a in range(2) for b in range(2) for c in range(2)}      # children of (0,1,0,0)
    want |= {(2, 4 + a, b, 2 + c) for a in range(2) for b in range(2) for c in range(2)}  # children of (1,2,0,1)
    assert got == want


# ------------------------------------------------------------------ helpers of the full-size parity tests
def test_census_classes_equals_the_plain_census(oracle):
    """psdo_census_classes (parallel, split by size class, optional tile window) against the plain
    serial psdo_census and a python recount of the class split, on a field that wraps around."""
    N, G = 8, 32
    pos = crossing_field(N, 2.0)
    c = oracle.census(pos, 1.0, G)
    f = oracle.census_classes(pos, 1.0, G)
    nt = G // 8
    assert np.array_equal((f["counts_small"] + f["counts_large"]).ravel(), c["tile_counts"])
    for k in ("hist_tet", "hist_pair"):
        assert np.array_equal(f[k], c[k])
    for k in ("n_tets", "n_pairs", "sum_cells", "max_cells", "n_inverted"):
        assert f[k] == c[k]
    # the class split: small = buckets 0..3 of hist_pair (<= 8 cells), per tile by a python recount
    assert int(f["counts_small"].sum()) == int(c["hist_pair"][:4].sum())
    small = np.zeros((nt, nt, nt), dtype=np.int64)
    for i in range(N):
        for j in range(N):
            for k in range(N):
                for t in range(6):
                    _, _, lo, hi = oracle.build_tet(pos, 1.0, G, i, j, k, t)
                    per_axis = []
                    for a in range(3):
                        d = {}
                        for cc in range(int(lo[a]), int(hi[a]) + 1):
                            d[(cc % G) // 8] = d.get((cc % G) // 8, 0) + 1
                        per_axis.append(d)
                    for tx, nx in per_axis[0].items():
                        for ty, ny in per_axis[1].items():
                            for tz, nz in per_axis[2].items():
                                small[tx, ty, tz] += nx * ny * nz <= 8
    assert np.array_equal(small, f["counts_small"].astype(np.int64))
    # a window of tiles that wraps around the box
    w = oracle.census_classes(pos, 1.0, G, win_lo=(3, 0, 2), win_n=(2, 4, 1))
    idx = np.ix_([3, 0], range(4), [2])
    assert np.array_equal(w["counts_small"], f["counts_small"][idx])
    assert np.array_equal(w["counts_large"], f["counts_large"][idx])
    assert w["n_pairs"] == int(w["counts_small"].sum() + w["counts_large"].sum()) == int(w["hist_pair"].sum())
    assert np.array_equal(w["hist_tet"], f["hist_tet"])
    # another threshold
    g = oracle.census_classes(pos, 1.0, G, small_max=64)
    assert int(g["counts_small"].sum()) == int(c["hist_pair"][:7].sum())


def test_deposit_windows_equals_single_windows(oracle):
    pos = crossing_field(6, 1.5)
    G = 12
    wins = [((10, 3, 0), (4, 5, 12)), ((0, 0, 0), (3, 3, 3)), ((11, 11, 11), (2, 2, 2))]
    many = oracle.deposit_windows(pos, 1.0, 1.0, G, wins)
    for (lo, n), got in zip(wins, many):
        assert np.allclose(got, oracle.deposit_window(pos, 1.0, 1.0, G, lo, n), rtol=1e-12, atol=1e-18)


def test_extreme_tets_against_a_python_scan(oracle):
    N, G = 8, 32
    pos = crossing_field(N, 2.5)
    e = oracle.extreme_tets(pos, 1.0, G, min_cells=8)
    best_n, best_thin, thin_tet = -1, np.inf, None
    for i in range(N):
        for j in range(N):
            for k in range(N):
                for t in range(6):
                    verts, det, lo, hi = oracle.build_tet(pos, 1.0, G, i, j, k, t)
                    n = int(np.prod(hi - lo + 1))
                    best_n = max(best_n, n)
                    g = verts * G
                    box = float(np.prod(g.max(0) - g.min(0)))
                    if n >= 8 and det != 0 and abs(det) / box < best_thin:
                        best_thin, thin_tet = abs(det) / box, (i, j, k, t)
    assert e["largest"]["n_cells"] == best_n
    i, j, k, t = e["largest"]["tet"]
    _, _, lo, hi = oracle.build_tet(pos, 1.0, G, i, j, k, t)
    assert int(np.prod(hi - lo + 1)) == best_n and np.array_equal(lo, e["largest"]["lo"])
    assert e["thinnest"]["tet"] == thin_tet and np.isclose(e["thinnest"]["ratio"], best_thin, rtol=1e-12)

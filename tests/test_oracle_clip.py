"""Pins for the oracle's tet-cube intersection (oracle/psd_oracle.c, O1/O3).

None of these re-types the oracle's algorithm (iterative plane splitting).
They check it against what the mathematics fixes: closed forms, invariants, exact rational
values and Monte Carlo.
"""
import itertools
from fractions import Fraction

import numpy as np
import pytest

CORNER_TET = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [0, 0, 1]], dtype=np.float64)


def corner_tet_orthant_volume(a, b, c):
    """vol({x,y,z>=0, x+y+z<=1} n [0,a]x[0,b]x[0,c]) by inclusion-exclusion of the three
    caps {x>a},{y>b},{z>c} of the simplex (each cap set is a scaled simplex):
    (1/6) sum_S (-1)^|S| (1 - sum_S)_+^3.  Works in Fractions or floats."""
    tot = 0
    for S in itertools.product((0, 1), repeat=3):
        s = S[0] * a + S[1] * b + S[2] * c
        r = 1 - s
        if r > 0:
            tot += (-1) ** sum(S) * r ** 3
    return tot / 6


def corner_tet_box_volume(lo, hi):
    """Any box: clamp to the octant, then 8-corner inclusion-exclusion of orthant volumes."""
    lo = [max(x, 0) for x in lo]
    hi = [max(x, 0) for x in hi]
    tot = 0
    for S in itertools.product((0, 1), repeat=3):
        p = [hi[i] if S[i] else lo[i] for i in range(3)]
        tot += (-1) ** (3 - sum(S)) * corner_tet_orthant_volume(*p)
    return tot


def test_kuhn_table_tiles_the_cube(oracle):
    """PAPER.md:45 '6 tetrahedra'; Q1.  dets = +1, volumes sum to 1, every random
    point of the cube is in exactly one tet, all six share the diagonal 0-7, and opposite cube
    faces carry the same diagonal (so neighbouring cells' tets share faces)."""
    K = oracle.kuhn_table()
    corners = np.array([[b & 1, (b >> 1) & 1, (b >> 2) & 1] for b in range(8)], dtype=np.float64)
    dets = []
    for t in K:
        v = corners[t]
        dets.append(np.linalg.det(v[1:] - v[0]))
        assert t[0] == 0 and t[3] == 7
    assert np.allclose(dets, 1.0)
    rng = np.random.default_rng(0)
    pts = rng.random((20000, 3))
    inside = np.zeros(len(pts), dtype=int)
    for t in K:
        v = corners[t]
        A = (v[1:] - v[0]).T
        lam = np.linalg.solve(A, (pts - v[0]).T).T
        l0 = 1 - lam.sum(axis=1)
        inside += ((lam > 0).all(axis=1) & (l0 > 0)).astype(int)
    assert (inside == 1).all()
    # face diagonals: the set of tet edges lying in face x=0 translated by +x equals that in x=1
    edges = set()
    for t in K:
        for a, b in itertools.combinations(t, 2):
            edges.add((min(a, b), max(a, b)))
    for ax in range(3):
        bit = 1 << ax
        lo = {(a, b) for a, b in edges if not a & bit and not b & bit}
        hi = {(a - bit, b - bit) for a, b in edges if a & bit and b & bit}
        assert lo == hi


def test_build_tet_matches_lattice_offsets(oracle):
    """O1: on an unperturbed lattice tet t of cell (i,j,k) has vertices q + corner offsets."""
    import psd_inputs
    N, G = 4, 8
    pos = psd_inputs.lattice(N, shift=(0.01, 0.02, 0.03))
    K = oracle.kuhn_table()
    for (i, j, k) in [(0, 0, 0), (3, 3, 3), (1, 3, 2)]:  # (3,3,3) wraps on every axis
        for t in range(6):
            v, det, lo, hi = oracle.build_tet(pos, 1.0, G, i, j, k, t)
            base = np.array([i, j, k]) / N + np.array([0.01, 0.02, 0.03])
            offs = np.array([[b & 1, (b >> 1) & 1, (b >> 2) & 1] for b in K[t]]) / N
            assert np.allclose(v, base + offs, atol=1e-15)
            assert np.isclose(det, (G / N) ** 3)


def test_corner_tet_exact_rational_boxes(oracle):
    """Closed form in exact rational arithmetic vs the oracle (double and gold)."""
    rng = np.random.default_rng(1)
    for _ in range(200):
        lo = [Fraction(int(rng.integers(-8, 24)), 32) for _ in range(3)]
        hi = [l + Fraction(int(rng.integers(1, 24)), 32) for l in lo]
        exact = corner_tet_box_volume(lo, hi)
        got = oracle.tet_aabox_volume(CORNER_TET, [float(x) for x in lo], [float(x) for x in hi])
        gold = oracle.tet_aabox_volume(CORNER_TET, [float(x) for x in lo], [float(x) for x in hi],
                                       kind="gold")
        assert abs(got - float(exact)) < 2e-16 + 1e-14 * float(exact)
        assert abs(gold - float(exact)) < 1e-17 + 1e-15 * float(exact)


def test_corner_tet_aligned_grid_golden(oracle):
    """tests/golden/corner_tet_aligned.txt: on an aligned n-grid cell (i,j,k) of the corner tet
    scaled by n holds 1/6, 5/6, 1, 0 of a cell for u = n-(i+j+k) = 1, 2, >=3, <=0."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "corner_tet_aligned.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    table = {int(r[0]): Fraction(r[1]) for r in rows}
    n = 5
    vol, V = oracle.tet_deposit_box(CORNER_TET * n, [0, 0, 0], [n, n, n])
    assert np.isclose(V, n ** 3 / 6)
    for i, j, k in itertools.product(range(n), repeat=3):
        u = n - (i + j + k)
        want = float(table[min(max(u, 0), 3)])
        assert abs(vol[i, j, k] - want) < 1e-14


def test_kuhn_tet_aligned_grid_golden(oracle):
    """tests/golden/kuhn_tet_aligned.txt: the Kuhn tet {x<=y<=z} of an n-cube on the aligned
    n-grid gives cell (i,j,k): 1 if i<j<k; 1/2 if exactly one equality; 1/6 if i=j=k; else 0."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "kuhn_tet_aligned.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    table = {r[0]: Fraction(r[1]) for r in rows}
    n = 4
    tet = np.array([[0, 0, 0], [0, 0, 1], [0, 1, 1], [1, 1, 1]], dtype=np.float64) * n  # x<=y<=z
    vol, _ = oracle.tet_deposit_box(tet, [0, 0, 0], [n, n, n])
    for i, j, k in itertools.product(range(n), repeat=3):
        if i < j < k:
            key = "strict"
        elif i == j == k:
            key = "all_equal"
        elif (i == j < k) or (i < j == k):
            key = "one_equal"
        else:
            key = "outside"
        assert abs(vol[i, j, k] - float(table[key])) < 1e-14, (i, j, k)


def random_tets(rng, n, scale=3.0):
    return rng.random((n, 4, 3)) * scale + rng.random((n, 1, 3)) * 2.0


def tet_volume(v):
    return abs(np.linalg.det(v[1:] - v[0])) / 6.0


def test_sum_over_cells_is_tet_volume(oracle):
    """Pin 3: sum_c vol(T n C_c) = |V_T|, including thin slivers."""
    rng = np.random.default_rng(2)
    tets = list(random_tets(rng, 60))
    for _ in range(40):  # slivers: 4th vertex almost in the plane of the other three
        v = random_tets(rng, 1, 6.0)[0]
        lam = rng.random(3)
        lam /= lam.sum()
        v[3] = lam @ v[:3] + rng.normal(size=3) * 10.0 ** rng.uniform(-9, -3)
        tets.append(v)
    for v in tets:
        lo = np.floor(v.min(axis=0)).astype(int)
        n = np.floor(v.max(axis=0)).astype(int) - lo + 1
        vol, V = oracle.tet_deposit_box(v, lo, n)
        # numpy's double determinant is the less accurate side on slivers (oracle: long double)
        assert np.isclose(V, tet_volume(v), rtol=1e-9, atol=2e-15 * np.abs(v).max() ** 3)
        assert (vol >= 0).all()
        assert abs(vol.sum() - V) <= 1e-12 * max(V, 1e-300) + 4e-16 * np.abs(v).max() ** 2


def curry_schoenberg_cdf(x, a):
    """Fraction of a simplex with vertex coordinates x (distinct) having coordinate < a:
    F(a) = 1 - sum_i (x_i - a)_+^3 / prod_{j != i} (x_i - x_j)."""
    tot = 0.0
    for i in range(4):
        d = x[i] - a
        if d > 0:
            den = 1.0
            for j in range(4):
                if j != i:
                    den *= x[i] - x[j]
            tot += d ** 3 / den
    return 1.0 - tot


def test_axis_marginals_match_bspline_cdf(oracle):
    """Pin 2: slab sums of the deposit equal the Curry-Schoenberg B-spline CDF differences."""
    rng = np.random.default_rng(3)
    for v in random_tets(rng, 40, 4.0):
        lo = np.floor(v.min(axis=0)).astype(int)
        n = np.floor(v.max(axis=0)).astype(int) - lo + 1
        vol, V = oracle.tet_deposit_box(v, lo, n)
        for ax in range(3):
            x = v[:, ax]
            if np.min(np.abs(x[:, None] - x[None, :]) + np.eye(4)) < 0.05:
                continue  # the closed form divides by coordinate differences
            other = tuple(a for a in range(3) if a != ax)
            slab = vol.sum(axis=other)
            for s in range(n[ax]):
                want = V * (curry_schoenberg_cdf(x, lo[ax] + s + 1) - curry_schoenberg_cdf(x, lo[ax] + s))
                assert abs(slab[s] - want) < 1e-9 * V + 1e-12


def test_invariances(oracle):
    """Pin 4: integer translations, axis permutations / reflections, vertex relabelling."""
    rng = np.random.default_rng(4)
    for v in random_tets(rng, 12, 2.5):
        lo = np.array([0.3, 0.7, 1.1])
        hi = lo + np.array([1.0, 0.8, 1.3])
        base = oracle.tet_aabox_volume(v, lo, hi)
        for perm in itertools.permutations(range(4)):
            assert np.isclose(oracle.tet_aabox_volume(v[list(perm)], lo, hi), base, rtol=1e-12, atol=1e-15)
        for ap in itertools.permutations(range(3)):
            ap = list(ap)
            assert np.isclose(oracle.tet_aabox_volume(v[:, ap], lo[ap], hi[ap]), base, rtol=1e-12, atol=1e-15)
        for ax in range(3):
            w = v.copy(); w[:, ax] *= -1
            l2, h2 = lo.copy(), hi.copy()
            l2[ax], h2[ax] = -hi[ax], -lo[ax]
            assert np.isclose(oracle.tet_aabox_volume(w, l2, h2), base, rtol=1e-12, atol=1e-15)
        sh = np.array([5.0, -3.0, 17.0])
        assert np.isclose(oracle.tet_aabox_volume(v + sh, lo + sh, hi + sh), base, rtol=1e-11, atol=1e-14)


def test_trivial_configurations(oracle):
    """PAPER.md:137 trivial cases: tet inside the cell -> |V|; cell inside the tet -> cell volume;
    disjoint -> 0; a vertex / face exactly on a cell plane (Q7)."""
    small = np.array([[0.2, 0.2, 0.2], [0.5, 0.2, 0.3], [0.3, 0.6, 0.2], [0.25, 0.3, 0.7]])
    assert np.isclose(oracle.tet_box_volume(small, [0, 0, 0], 1.0), tet_volume(small), rtol=1e-13)
    big = np.array([[-10, -10, -10], [30, -10, -10], [-10, 30, -10], [-10, -10, 30]], dtype=float)
    assert np.isclose(oracle.tet_box_volume(big, [0, 0, 0], 1.0), 1.0, rtol=1e-13)
    assert oracle.tet_box_volume(small, [1, 0, 0], 1.0) == 0.0
    assert oracle.tet_box_volume(small, [-1, 0, 0], 1.0) == 0.0
    # unit corner tet touches the cell x in [1,2] only in one point
    assert oracle.tet_box_volume(CORNER_TET, [1, 0, 0], 1.0) == 0.0
    # all vertices on cell planes: the cube's Kuhn tets fill 1/6 each
    K = oracle.kuhn_table()
    corners = np.array([[b & 1, (b >> 1) & 1, (b >> 2) & 1] for b in range(8)], dtype=np.float64)
    for t in K:
        assert np.isclose(oracle.tet_box_volume(corners[t], [0, 0, 0], 1.0), 1 / 6, rtol=1e-14)


def test_monte_carlo(oracle):
    """Pin 5: uniform samples in the tet binned to cells (gross-error check)."""
    rng = np.random.default_rng(5)
    ns = 400000
    for v in random_tets(rng, 4, 3.0):
        e = -np.log(rng.random((ns, 4)))
        lam = e / e.sum(axis=1, keepdims=True)  # uniform on the simplex
        pts = lam @ v
        lo = np.floor(v.min(axis=0)).astype(int)
        n = np.floor(v.max(axis=0)).astype(int) - lo + 1
        idx = np.floor(pts).astype(int) - lo
        hist = np.zeros(n)
        np.add.at(hist, (idx[:, 0], idx[:, 1], idx[:, 2]), 1.0)
        vol, V = oracle.tet_deposit_box(v, lo, n)
        frac = vol / V
        sigma = np.sqrt(np.maximum(frac * (1 - frac), 1e-6) / ns)
        assert (np.abs(hist / ns - frac) < 6 * sigma + 1e-5).all()


def test_gold_agrees_with_double_on_slivers(oracle):
    """Pin 7: __float128 geometry vs double on hand-made slivers sets the error budget."""
    rng = np.random.default_rng(6)
    worst = 0.0
    for _ in range(60):
        v = random_tets(rng, 1, 40.0)[0]
        lam = rng.random(3); lam /= lam.sum()
        v[3] = lam @ v[:3] + rng.normal(size=3) * 10.0 ** rng.uniform(-6, -2)
        lo = np.floor(v.min(axis=0)).astype(int)
        n = np.minimum(np.floor(v.max(axis=0)).astype(int) - lo + 1, 6)
        d, Vd = oracle.tet_deposit_box(v, lo, n)
        g, Vg = oracle.tet_deposit_box(v, lo, n, kind="gold")
        assert np.isclose(Vd, Vg, rtol=1e-12)
        err = np.abs(d - g).max() / Vg
        worst = max(worst, err)
    # relative to the tet volume (= relative mass error), far inside the 1e-6 parity budget
    assert worst < 1e-8, worst

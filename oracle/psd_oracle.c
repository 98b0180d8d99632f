/*
 * psd_oracle.c -- TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct CPU
 * implementation of the phase-space-element mass deposit of
 *   R. Kaehler, "Massively Parallel Computation of Accurate Densities for N-body
 *   Dark Matter Simulations using the Phase-Space-Element Method" (arXiv:1612.09491),
 * written from the paper text (/root/reference/PAPER.md, cited as PAPER.md:LINE).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call this.  It shares NO code, header, table or constant with the CUDA
 * path under paper_1612_09491_b200/ and neither side includes the other.
 *
 * What it computes (Eq. 1 integrated over a cell; "the
 * resulting volume is transformed to its mass equivalent"):
 *
 *     mass[c] = sum over all 6 N^3 tets T (and periodic images) of
 *               m * vol(T n C_c) / |vol(T)|,          m = M / (6 N^3)
 *
 * How: the paper's own route.
 *   O1  PAPER.md:39-45  Lagrangian cell (i,j,k) -> 8 corner particles (indices mod N),
 *       minimum-image unwrap relative to corner 0, 6 tetrahedra per cell (Kuhn split,
 *       DESIGN.md reading Q1), equal mass per tet.
 *   O2  PAPER.md:137    axis-aligned bounding box of the tet -> integer cell range.
 *   O3  PAPER.md:155-159 (section 6.3) tet-cube intersection by ITERATIVE PLANE
 *       SPLITTING: the tet is split against the 6 face planes of the cell one at a
 *       time, the kept part is re-tetrahedralised (the paper's look-up table, written
 *       here as its 5 topological cases), the volume is the sum of the leaf tets.
 *       No trivial-case shortcuts, no complement trick:
 *       they do not change the result.
 *   O4  PAPER.md:137    mass += m * vol / V  into the (periodic) cell.
 *   O5  counters compared bit-exactly with the GPU census (tile = 8^3 cells).
 *   O6  PAPER.md:72     patch deposit: same as O2-O4 on the level grid, restricted to
 *       the patch's P^3 box.   PAPER.md:66: refinement by tet count.
 *   O7  PAPER.md:74-76  (section 4, Fig. 4) memory-lean refinement census: the Lagrangian
 *       grid is cut into sub-blocks of B^3 cells, each sub-block's minimal axis-aligned
 *       bounding box is taken, and the number of tets over a tree node is ESTIMATED as
 *       (tets of the sub-block) x vol(box n node) / vol(box), summed over sub-blocks
 *       (psdo_subblock_counts; reading Q17 for the fixed-point unit).
 *
 * Precision: REAL is double (the timed baseline) or __float128 ("gold", -DPSDO_GOLD)
 * for the geometry; sums into the output grid are always double.  The tet determinant
 * is evaluated in long double (>= 64-bit mantissa on x86) in the double build so that
 * the denominator |V| of a sliver tet is not the limiting error (reading Q5b).
 *
 * Compile with -ffp-contract=off: the integer cell ranges (O2, O5) must come from
 * individually rounded IEEE operations so that they can be compared bit-exactly.
 *
 * parity pins: tests/test_oracle_*.py (closed forms, invariants, Monte Carlo, rational
 * golden values) -- none of them re-types these formulas.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifdef PSDO_GOLD
#include <quadmath.h>
typedef __float128 REAL;
typedef __float128 DETREAL;
#define R_FLOOR floorq
#define R_RINT rintq
#define R_FABS fabsq
#elif defined(PSDO_SINGLE)
/* the geometry (unwrap, scaling, splitting, leaf volumes) in fp32, determinant and sums in fp64:
 * exists only to measure whether an fp32 clip could hold the parity tolerance (it does not;
 * DESIGN.md section 4 item 4, tests/test_oracle_deposit.py) */
typedef float REAL;
typedef double DETREAL;
#define R_FLOOR floorf
#define R_RINT rintf
#define R_FABS fabsf
#else
typedef double REAL;
typedef long double DETREAL;
#define R_FLOOR floor
#define R_RINT rint
#define R_FABS fabs
#endif

#define PSDO_F32 0
#define PSDO_F64 1
#define PSDO_MODE_MASS 0   /* weight m/|V|                      */
#define PSDO_MODE_SIGNED 1 /* weight sign(det): every cell -> 1 */

/* ---- O1: Kuhn / Freudenthal split (Q1).  Corner index b = dx + 2 dy + 4 dz.
 * All six share the main diagonal 0-7; one tet per monotone lattice path.           */
static const int KUHN[6][4] = {
    {0, 1, 3, 7}, {0, 5, 1, 7}, {0, 3, 2, 7}, {0, 2, 6, 7}, {0, 4, 5, 7}, {0, 6, 4, 7}};

typedef struct {
    const void *pos;
    int dtype, stride, N;
    double L;
} particles_t;

static inline REAL load_coord(const particles_t *p, int64_t idx, int c) {
    if (p->dtype == PSDO_F32) return (REAL)((const float *)p->pos)[idx * p->stride + c];
    return (REAL)((const double *)p->pos)[idx * p->stride + c];
}

/* 8 unwrapped corners of Lagrangian cell (i,j,k), in box units. */
static void cell_corners(const particles_t *p, int i, int j, int k, REAL P[8][3]) {
    const int N = p->N;
    const REAL L = (REAL)p->L;
    for (int b = 0; b < 8; ++b) {
        int ii = (i + (b & 1)) % N, jj = (j + ((b >> 1) & 1)) % N, kk = (k + ((b >> 2) & 1)) % N;
        int64_t idx = ((int64_t)ii * N + jj) * N + kk;
        for (int c = 0; c < 3; ++c) P[b][c] = load_coord(p, idx, c);
    }
    for (int b = 1; b < 8; ++b)
        for (int c = 0; c < 3; ++c) {
            REAL d = P[b][c] - P[0][c];
            REAL q = d / L;
            REAL r = R_RINT(q);
            REAL s = L * r;
            P[b][c] = P[b][c] - s; /* minimum image of corner 0 (Q3, Q4) */
        }
}

static DETREAL det3(const REAL v[4][3]) {
    DETREAL a[3], b[3], c[3];
    for (int x = 0; x < 3; ++x) {
        a[x] = (DETREAL)v[1][x] - (DETREAL)v[0][x];
        b[x] = (DETREAL)v[2][x] - (DETREAL)v[0][x];
        c[x] = (DETREAL)v[3][x] - (DETREAL)v[0][x];
    }
    return a[0] * (b[1] * c[2] - b[2] * c[1]) - a[1] * (b[0] * c[2] - b[2] * c[0]) +
           a[2] * (b[0] * c[1] - b[1] * c[0]);
}

/* ---- O3: PAPER.md:155-159.  Planes of the unit cell [0,1]^3 in the order
 * x>=0, x<=1, y>=0, y<=1, z>=0, z<=1.  Signed distance, inside is d >= 0 (Q7).       */
static inline REAL plane_dist(const REAL *v, int plane) {
    int ax = plane >> 1;
    return (plane & 1) ? ((REAL)1 - v[ax]) : v[ax];
}

/* point where edge a->b meets the plane; only called with da >= 0 > db. */
static inline void edge_cut(const REAL *a, const REAL *b, REAL da, REAL db, REAL *out) {
    REAL t = da / (da - db);
    for (int c = 0; c < 3; ++c) out[c] = a[c] + t * (b[c] - a[c]);
}

static REAL tet_vol_abs(const REAL v[4][3]) {
    REAL a[3], b[3], c[3];
    for (int x = 0; x < 3; ++x) {
        a[x] = v[1][x] - v[0][x];
        b[x] = v[2][x] - v[0][x];
        c[x] = v[3][x] - v[0][x];
    }
    REAL d = a[0] * (b[1] * c[2] - b[2] * c[1]) - a[1] * (b[0] * c[2] - b[2] * c[0]) +
             a[2] * (b[0] * c[1] - b[1] * c[0]);
    return R_FABS(d) / (REAL)6;
}

/* prism with triangles (a,b,c) and (a2,b2,c2), side edges a-a2, b-b2, c-c2, planar
 * side quads: staircase split into 3 tets. */
static REAL split_clip(const REAL tet[4][3], int plane);

static REAL prism_clip(const REAL *a, const REAL *b, const REAL *c, const REAL *a2, const REAL *b2,
                       const REAL *c2, int plane) {
    REAL t[4][3];
    REAL s = 0;
    memcpy(t[0], a, sizeof(REAL) * 3); memcpy(t[1], b, sizeof(REAL) * 3);
    memcpy(t[2], c, sizeof(REAL) * 3); memcpy(t[3], a2, sizeof(REAL) * 3);
    s += split_clip(t, plane);
    memcpy(t[0], a2, sizeof(REAL) * 3); memcpy(t[1], b, sizeof(REAL) * 3);
    memcpy(t[2], c, sizeof(REAL) * 3); memcpy(t[3], b2, sizeof(REAL) * 3);
    s += split_clip(t, plane);
    memcpy(t[0], a2, sizeof(REAL) * 3); memcpy(t[1], b2, sizeof(REAL) * 3);
    memcpy(t[2], c, sizeof(REAL) * 3); memcpy(t[3], c2, sizeof(REAL) * 3);
    s += split_clip(t, plane);
    return s;
}

/* volume of tet n {planes plane..5 of the unit cell} */
static REAL split_clip(const REAL tet[4][3], int plane) {
    if (plane == 6) return tet_vol_abs(tet);
    REAL d[4];
    int in[4], nin = 0;
    for (int v = 0; v < 4; ++v) {
        d[v] = plane_dist(tet[v], plane);
        in[v] = d[v] >= 0;
        nin += in[v];
    }
    if (nin == 4) return split_clip(tet, plane + 1);
    if (nin == 0) return 0;
    int vi[4], vo[4], ni = 0, no = 0; /* inside / outside vertex lists */
    for (int v = 0; v < 4; ++v) {
        if (in[v]) vi[ni++] = v; else vo[no++] = v;
    }
    if (nin == 1) { /* small tet at the inside vertex */
        int A = vi[0];
        REAL t[4][3];
        memcpy(t[0], tet[A], sizeof(REAL) * 3);
        for (int q = 0; q < 3; ++q) edge_cut(tet[A], tet[vo[q]], d[A], d[vo[q]], t[q + 1]);
        return split_clip(t, plane + 1);
    }
    if (nin == 3) { /* prism: 3 inside vertices + 3 cuts on the edges to the outside vertex */
        int O = vo[0];
        REAL c[3][3];
        for (int q = 0; q < 3; ++q) edge_cut(tet[vi[q]], tet[O], d[vi[q]], d[O], c[q]);
        return prism_clip(tet[vi[0]], tet[vi[1]], tet[vi[2]], c[0], c[1], c[2], plane + 1);
    }
    /* nin == 2: wedge = prism with triangles (A, AC, AD) and (B, BC, BD) */
    {
        int A = vi[0], B = vi[1], C = vo[0], D = vo[1];
        REAL ac[3], ad[3], bc[3], bd[3];
        edge_cut(tet[A], tet[C], d[A], d[C], ac);
        edge_cut(tet[A], tet[D], d[A], d[D], ad);
        edge_cut(tet[B], tet[C], d[B], d[C], bc);
        edge_cut(tet[B], tet[D], d[B], d[D], bd);
        return prism_clip(tet[A], ac, ad, tet[B], bc, bd, plane + 1);
    }
}

/* vol(T n unit cell at integer corner c) with T in grid units: shift to cell-local first */
static REAL tet_cell_volume(const REAL g[4][3], const int64_t c[3]) {
    REAL t[4][3];
    for (int v = 0; v < 4; ++v)
        for (int x = 0; x < 3; ++x) t[v][x] = g[v][x] - (REAL)c[x];
    return split_clip(t, 0);
}

/* ---- one tet prepared for deposit on a grid with G cells per side ---- */
typedef struct {
    REAL g[4][3];      /* vertices in grid units (cells), unwrapped */
    int64_t lo[3], hi[3]; /* O2: integer cell range, unwrapped       */
    DETREAL det;       /* signed 6*volume in grid units            */
} tet_t;

static void make_tet(const REAL P[8][3], int t, REAL scale, tet_t *out) {
    for (int v = 0; v < 4; ++v)
        for (int x = 0; x < 3; ++x) out->g[v][x] = P[KUHN[t][v]][x] * scale;
    for (int x = 0; x < 3; ++x) {
        REAL mn = out->g[0][x], mx = out->g[0][x];
        for (int v = 1; v < 4; ++v) {
            if (out->g[v][x] < mn) mn = out->g[v][x];
            if (out->g[v][x] > mx) mx = out->g[v][x];
        }
        out->lo[x] = (int64_t)R_FLOOR(mn);
        out->hi[x] = (int64_t)R_FLOOR(mx);
    }
    out->det = det3(out->g);
}

static inline int64_t wrap(int64_t c, int64_t G) { return ((c % G) + G) % G; }

/* target of a deposit: either the whole periodic G^3 grid, or a box window of it
 * (wrapped coordinates win_lo <= c < win_lo+win_n per axis, stored densely).        */
typedef struct {
    int64_t G;
    double *out;
    int windowed;
    int64_t wlo[3], wn[3];
} target_t;

static inline double *target_cell(const target_t *T, int64_t cx, int64_t cy, int64_t cz) {
    int64_t w[3] = {wrap(cx, T->G), wrap(cy, T->G), wrap(cz, T->G)};
    if (!T->windowed) return T->out + (w[0] * T->G + w[1]) * T->G + w[2];
    int64_t r[3];
    for (int x = 0; x < 3; ++x) {
        r[x] = wrap(w[x] - T->wlo[x], T->G);
        if (r[x] >= T->wn[x]) return NULL;
    }
    return T->out + (r[0] * T->wn[1] + r[1]) * T->wn[2] + r[2];
}

/* does the (unwrapped) range [lo,hi] meet the window along one axis? */
static int range_meets_window(int64_t lo, int64_t hi, int64_t G, int64_t wlo, int64_t wn) {
    if (hi - lo + 1 >= G) return 1;
    int64_t r = wrap(lo - wlo, G); /* position of lo relative to window start */
    if (r < wn) return 1;
    return r + (hi - lo) >= G; /* wraps around into the window */
}

static void deposit_tet(const tet_t *t, double m, int mode, const target_t *T, int64_t *n_cand,
                        int64_t *n_nonzero, int64_t *n_degenerate) {
    if (T->windowed) {
        for (int x = 0; x < 3; ++x)
            if (!range_meets_window(t->lo[x], t->hi[x], T->G, T->wlo[x], T->wn[x])) return;
    }
    DETREAL det = t->det;
    if (det == 0) { /* Q6: degenerate tet -> all mass to the cell holding the centroid */
        if (n_degenerate) ++*n_degenerate;
        if (mode != PSDO_MODE_MASS) return;
        int64_t c[3];
        for (int x = 0; x < 3; ++x)
            c[x] = (int64_t)R_FLOOR((t->g[0][x] + t->g[1][x] + t->g[2][x] + t->g[3][x]) / (REAL)4);
        double *cell = target_cell(T, c[0], c[1], c[2]);
        if (cell) {
#pragma omp atomic
            *cell += m;
        }
        return;
    }
    REAL V = (REAL)((det < 0 ? -det : det) / (DETREAL)6);
    REAL w = (mode == PSDO_MODE_MASS) ? (REAL)m / V : (det < 0 ? (REAL)-1 : (REAL)1);
    for (int64_t cx = t->lo[0]; cx <= t->hi[0]; ++cx)
        for (int64_t cy = t->lo[1]; cy <= t->hi[1]; ++cy)
            for (int64_t cz = t->lo[2]; cz <= t->hi[2]; ++cz) {
                double *cell = target_cell(T, cx, cy, cz);
                if (!cell) continue; /* outside the window / patch */
                if (n_cand) ++*n_cand;
                int64_t c[3] = {cx, cy, cz};
                REAL vol = tet_cell_volume(t->g, c);
                if (vol != 0 && n_nonzero) ++*n_nonzero;
                double add = (double)(w * vol);
#pragma omp atomic
                *cell += add;
            }
}

/* ===================================================================== exported */

/* stats[0]=n_tets, [1]=sum of AABB cells (candidates), [2]=cells with vol != 0,
 * [3]=degenerate tets, [4]=tets with det < 0 (inverted).                        */
static int deposit_common(const void *pos, int dtype, int stride, int N, double L, double M, int G,
                          const target_t *T, int mode, int64_t *stats) {
    if (N < 2 || G < 1 || !(L > 0) || (stride != 3 && stride != 4)) return 1;
    particles_t p = {pos, dtype, stride, N, L};
    const double m = M / (6.0 * (double)N * (double)N * (double)N);
    const REAL scale = (REAL)G / (REAL)L;
    int64_t s_cand = 0, s_nz = 0, s_deg = 0, s_inv = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : s_cand, s_nz, s_deg, s_inv)
    for (int i = 0; i < N; ++i)
        for (int j = 0; j < N; ++j)
            for (int k = 0; k < N; ++k) {
                REAL P[8][3];
                cell_corners(&p, i, j, k, P);
                for (int t = 0; t < 6; ++t) {
                    tet_t tet;
                    make_tet(P, t, scale, &tet);
                    if (tet.det < 0) ++s_inv;
                    deposit_tet(&tet, m, mode, T, &s_cand, &s_nz, &s_deg);
                }
            }
    if (stats) {
        stats[0] = (int64_t)6 * N * N * N;
        stats[1] = s_cand;
        stats[2] = s_nz;
        stats[3] = s_deg;
        stats[4] = s_inv;
    }
    return 0;
}

int psdo_deposit_uniform(const void *pos, int dtype, int stride, int N, double L, double M, int G,
                         double *grid, int mode, int64_t *stats) {
    target_t T = {G, grid, 0, {0, 0, 0}, {0, 0, 0}};
    memset(grid, 0, sizeof(double) * (size_t)G * G * G);
    return deposit_common(pos, dtype, stride, N, L, M, G, &T, mode, stats);
}

/* Deposit only into the window of cells win_lo[x] <= c < win_lo[x]+win_n[x] (wrapped);
 * out has win_n[0]*win_n[1]*win_n[2] entries.  Used to check a full-size run on
 * sampled regions: every tet is still visited, only its cells outside are skipped. */
int psdo_deposit_window(const void *pos, int dtype, int stride, int N, double L, double M, int G,
                        const int64_t *win_lo, const int64_t *win_n, double *out, int mode,
                        int64_t *stats) {
    target_t T = {G, out, 1, {win_lo[0], win_lo[1], win_lo[2]}, {win_n[0], win_n[1], win_n[2]}};
    for (int x = 0; x < 3; ++x)
        if (win_n[x] < 1 || win_n[x] > G) return 1;
    memset(out, 0, sizeof(double) * (size_t)(win_n[0] * win_n[1] * win_n[2]));
    return deposit_common(pos, dtype, stride, N, L, M, G, &T, mode, stats);
}

/* Same, restricted to Lagrangian cells with flat index in [cell_begin, cell_end):
 * the bounded sample that bench.py times (cpu_baseline). */
int psdo_deposit_uniform_range(const void *pos, int dtype, int stride, int N, double L, double M,
                               int G, double *grid, int mode, int64_t cell_begin, int64_t cell_end,
                               int64_t *stats) {
    if (N < 2 || G < 1 || !(L > 0) || (stride != 3 && stride != 4)) return 1;
    target_t T = {G, grid, 0, {0, 0, 0}, {0, 0, 0}};
    particles_t p = {pos, dtype, stride, N, L};
    const double m = M / (6.0 * (double)N * (double)N * (double)N);
    const REAL scale = (REAL)G / (REAL)L;
    int64_t s_cand = 0, s_nz = 0, s_deg = 0, s_inv = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : s_cand, s_nz, s_deg, s_inv)
    for (int64_t c = cell_begin; c < cell_end; ++c) {
        int k = (int)(c % N), j = (int)((c / N) % N), i = (int)(c / ((int64_t)N * N));
        REAL P[8][3];
        cell_corners(&p, i, j, k, P);
        for (int t = 0; t < 6; ++t) {
            tet_t tet;
            make_tet(P, t, scale, &tet);
            if (tet.det < 0) ++s_inv;
            deposit_tet(&tet, m, mode, &T, &s_cand, &s_nz, &s_deg);
        }
    }
    if (stats) {
        stats[0] = 6 * (cell_end - cell_begin);
        stats[1] = s_cand; stats[2] = s_nz; stats[3] = s_deg; stats[4] = s_inv;
    }
    return 0;
}

/* ---- O5: census.  tile = `tile`^3 cells (8).  For every tet: its AABB cell range
 * [lo,hi]; n_cells = prod(hi-lo+1); bucket b = bit_width(n_cells-1).
 *   tile_counts[(tx*nt+ty)*nt+tz] += 1 for every distinct periodic tile met;
 *   hist_tet[b] += 1;  hist_pair[b'] += 1 per (tet,tile) pair with b' from the number
 *   of the tet's range cells that fall in that tile (all images summed).
 * out_scalars: [0]=n_tets [1]=n_pairs [2]=sum n_cells [3]=max n_cells [4]=inverted  */
static inline int bit_width_u64(uint64_t v) {
    int b = 0;
    while (v) { ++b; v >>= 1; }
    return b;
}

int psdo_census(const void *pos, int dtype, int stride, int N, double L, int G, int tile,
                uint32_t *tile_counts, uint64_t *hist_tet, uint64_t *hist_pair,
                int64_t *out_scalars) {
    if (N < 2 || G < 1 || tile < 1 || G % tile) return 1;
    particles_t p = {pos, dtype, stride, N, L};
    const REAL scale = (REAL)G / (REAL)L;
    const int64_t nt = G / tile;
    memset(tile_counts, 0, sizeof(uint32_t) * (size_t)(nt * nt * nt));
    memset(hist_tet, 0, sizeof(uint64_t) * 64);
    memset(hist_pair, 0, sizeof(uint64_t) * 64);
    int64_t n_pairs = 0, sum_cells = 0, max_cells = 0, n_inv = 0;
    /* serial on purpose: plain counters, no atomics to reason about */
    for (int i = 0; i < N; ++i)
        for (int j = 0; j < N; ++j)
            for (int k = 0; k < N; ++k) {
                REAL P[8][3];
                cell_corners(&p, i, j, k, P);
                for (int t = 0; t < 6; ++t) {
                    tet_t tet;
                    make_tet(P, t, scale, &tet);
                    if (tet.det < 0) ++n_inv;
                    int64_t n[3], ncell = 1;
                    for (int x = 0; x < 3; ++x) { n[x] = tet.hi[x] - tet.lo[x] + 1; ncell *= n[x]; }
                    sum_cells += ncell;
                    if (ncell > max_cells) max_cells = ncell;
                    hist_tet[bit_width_u64((uint64_t)(ncell - 1))]++;
                    /* per axis: for each periodic tile index, how many range cells fall in it */
                    int64_t *cnt[3];
                    for (int x = 0; x < 3; ++x) {
                        cnt[x] = (int64_t *)calloc((size_t)nt, sizeof(int64_t));
                        for (int64_t c = tet.lo[x]; c <= tet.hi[x]; ++c) cnt[x][wrap(c, G) / tile]++;
                    }
                    for (int64_t tx = 0; tx < nt; ++tx) {
                        if (!cnt[0][tx]) continue;
                        for (int64_t ty = 0; ty < nt; ++ty) {
                            if (!cnt[1][ty]) continue;
                            for (int64_t tz = 0; tz < nt; ++tz) {
                                if (!cnt[2][tz]) continue;
                                tile_counts[(tx * nt + ty) * nt + tz]++;
                                ++n_pairs;
                                uint64_t inside = (uint64_t)(cnt[0][tx] * cnt[1][ty] * cnt[2][tz]);
                                hist_pair[bit_width_u64(inside - 1)]++;
                            }
                        }
                    }
                    for (int x = 0; x < 3; ++x) free(cnt[x]);
                }
            }
    out_scalars[0] = (int64_t)6 * N * N * N;
    out_scalars[1] = n_pairs;
    out_scalars[2] = sum_cells;
    out_scalars[3] = max_cells;
    out_scalars[4] = n_inv;
    return 0;
}

/* ---- O5 at full size: the same census, over Lagrangian slabs in parallel (per-thread
 * counters, summed at the end: integer work, order free), split by the a3 size class of the
 * pair (cells of the tet's range inside the tile <= small_max: "small", else "large"), and
 * optionally restricted to a window of tiles win_lo[x] <= t < win_lo[x] + win_n[x] (wrapped
 * tile coordinates; counts_small / counts_large are then dense over the window, hist_pair
 * and n_pairs cover the window's pairs only; hist_tet and the other scalars all tets).
 * Pinned against psdo_census (tests/test_oracle_deposit.py).                              */
int psdo_census_classes(const void *pos, int dtype, int stride, int N, double L, int G, int tile,
                        int64_t small_max, const int64_t *win_lo, const int64_t *win_n,
                        uint32_t *counts_small, uint32_t *counts_large, uint64_t *hist_tet,
                        uint64_t *hist_pair, int64_t *out_scalars) {
    if (N < 2 || G < 1 || tile < 1 || G % tile) return 1;
    particles_t p = {pos, dtype, stride, N, L};
    const REAL scale = (REAL)G / (REAL)L;
    const int64_t nt = G / tile;
    int64_t wlo[3] = {0, 0, 0}, wn[3] = {nt, nt, nt};
    if (win_lo && win_n)
        for (int x = 0; x < 3; ++x) {
            wlo[x] = win_lo[x]; wn[x] = win_n[x];
            if (wn[x] < 1 || wn[x] > nt) return 1;
        }
    const size_t nout = (size_t)(wn[0] * wn[1] * wn[2]);
    memset(counts_small, 0, sizeof(uint32_t) * nout);
    memset(counts_large, 0, sizeof(uint32_t) * nout);
    memset(hist_tet, 0, sizeof(uint64_t) * 64);
    memset(hist_pair, 0, sizeof(uint64_t) * 64);
    int64_t n_pairs = 0, sum_cells = 0, max_cells = 0, n_inv = 0;
    int failed = 0;
#pragma omp parallel
    {
        uint32_t *cs = (uint32_t *)calloc(nout, sizeof(uint32_t));
        uint32_t *cl = (uint32_t *)calloc(nout, sizeof(uint32_t));
        int64_t *cnt[3];
        for (int x = 0; x < 3; ++x) cnt[x] = (int64_t *)calloc((size_t)nt, sizeof(int64_t));
        uint64_t ht[64], hp[64];
        memset(ht, 0, sizeof ht);
        memset(hp, 0, sizeof hp);
        int64_t t_pairs = 0, t_sum = 0, t_max = 0, t_inv = 0;
        int ok = cs && cl && cnt[0] && cnt[1] && cnt[2];
        if (!ok) {
#pragma omp atomic write
            failed = 1;
        }
#pragma omp for schedule(dynamic, 1)
        for (int i = 0; i < N; ++i) {
            if (!ok) continue;
            for (int j = 0; j < N; ++j)
                for (int k = 0; k < N; ++k) {
                    REAL P[8][3];
                    cell_corners(&p, i, j, k, P);
                    for (int t = 0; t < 6; ++t) {
                        tet_t tet;
                        make_tet(P, t, scale, &tet);
                        if (tet.det < 0) ++t_inv;
                        int64_t ncell = 1;
                        for (int x = 0; x < 3; ++x) ncell *= tet.hi[x] - tet.lo[x] + 1;
                        t_sum += ncell;
                        if (ncell > t_max) t_max = ncell;
                        ht[bit_width_u64((uint64_t)(ncell - 1))]++;
                        for (int x = 0; x < 3; ++x)
                            for (int64_t c = tet.lo[x]; c <= tet.hi[x]; ++c) cnt[x][wrap(c, G) / tile]++;
                        /* the distinct tiles per axis: those of the cells of the range */
                        for (int64_t cx = tet.lo[0]; cx <= tet.hi[0]; ++cx) {
                            int64_t tx = wrap(cx, G) / tile;
                            if (cnt[0][tx] <= 0) continue; /* already visited (marked below) */
                            int64_t nx = cnt[0][tx];
                            cnt[0][tx] = -nx;
                            int64_t rx = wrap(tx - wlo[0], nt);
                            if (rx >= wn[0]) continue;
                            for (int64_t cy = tet.lo[1]; cy <= tet.hi[1]; ++cy) {
                                int64_t ty = wrap(cy, G) / tile;
                                if (cnt[1][ty] <= 0) continue;
                                int64_t ny = cnt[1][ty];
                                cnt[1][ty] = -ny;
                                int64_t ry = wrap(ty - wlo[1], nt);
                                if (ry >= wn[1]) continue;
                                for (int64_t cz = tet.lo[2]; cz <= tet.hi[2]; ++cz) {
                                    int64_t tz = wrap(cz, G) / tile;
                                    if (cnt[2][tz] <= 0) continue;
                                    int64_t nz = cnt[2][tz];
                                    cnt[2][tz] = -nz;
                                    int64_t rz = wrap(tz - wlo[2], nt);
                                    if (rz >= wn[2]) continue;
                                    uint64_t inside = (uint64_t)(nx * ny * nz);
                                    size_t o = (size_t)((rx * wn[1] + ry) * wn[2] + rz);
                                    if ((int64_t)inside <= small_max) cs[o]++; else cl[o]++;
                                    ++t_pairs;
                                    hp[bit_width_u64(inside - 1)]++;
                                }
                                for (int64_t cz = tet.lo[2]; cz <= tet.hi[2]; ++cz) { /* unmark z */
                                    int64_t tz = wrap(cz, G) / tile;
                                    if (cnt[2][tz] < 0) cnt[2][tz] = -cnt[2][tz];
                                }
                            }
                            for (int64_t cy = tet.lo[1]; cy <= tet.hi[1]; ++cy) { /* unmark y */
                                int64_t ty = wrap(cy, G) / tile;
                                if (cnt[1][ty] < 0) cnt[1][ty] = -cnt[1][ty];
                            }
                        }
                        for (int x = 0; x < 3; ++x) /* clear the touched entries */
                            for (int64_t c = tet.lo[x]; c <= tet.hi[x]; ++c) cnt[x][wrap(c, G) / tile] = 0;
                    }
                }
        }
#pragma omp critical
        {
            if (ok) {
                for (size_t o = 0; o < nout; ++o) { counts_small[o] += cs[o]; counts_large[o] += cl[o]; }
                for (int b = 0; b < 64; ++b) { hist_tet[b] += ht[b]; hist_pair[b] += hp[b]; }
                n_pairs += t_pairs; sum_cells += t_sum; n_inv += t_inv;
                if (t_max > max_cells) max_cells = t_max;
            }
        }
        free(cs); free(cl);
        for (int x = 0; x < 3; ++x) free(cnt[x]);
    }
    if (failed) return 2;
    out_scalars[0] = (int64_t)6 * N * N * N;
    out_scalars[1] = n_pairs;
    out_scalars[2] = sum_cells;
    out_scalars[3] = max_cells;
    out_scalars[4] = n_inv;
    return 0;
}

/* Deposit into K windows of the grid in one pass over the tets (the windows of psdo_deposit_window;
 * out holds them one after the other, window w has win_n[3w]*win_n[3w+1]*win_n[3w+2] entries). */
int psdo_deposit_windows(const void *pos, int dtype, int stride, int N, double L, double M, int G,
                         int K, const int64_t *win_lo, const int64_t *win_n, double *out, int mode) {
    if (N < 2 || G < 1 || !(L > 0) || (stride != 3 && stride != 4) || K < 1 || K > 64) return 1;
    target_t T[64];
    size_t off = 0;
    for (int w = 0; w < K; ++w) {
        for (int x = 0; x < 3; ++x)
            if (win_n[3 * w + x] < 1 || win_n[3 * w + x] > G) return 1;
        target_t t = {G, out + off, 1, {win_lo[3 * w], win_lo[3 * w + 1], win_lo[3 * w + 2]},
                      {win_n[3 * w], win_n[3 * w + 1], win_n[3 * w + 2]}};
        T[w] = t;
        off += (size_t)(win_n[3 * w] * win_n[3 * w + 1] * win_n[3 * w + 2]);
    }
    memset(out, 0, sizeof(double) * off);
    particles_t p = {pos, dtype, stride, N, L};
    const double m = M / (6.0 * (double)N * (double)N * (double)N);
    const REAL scale = (REAL)G / (REAL)L;
#pragma omp parallel for schedule(dynamic, 1)
    for (int i = 0; i < N; ++i)
        for (int j = 0; j < N; ++j)
            for (int k = 0; k < N; ++k) {
                REAL P[8][3];
                cell_corners(&p, i, j, k, P);
                for (int t = 0; t < 6; ++t) {
                    tet_t tet;
                    make_tet(P, t, scale, &tet);
                    for (int w = 0; w < K; ++w) deposit_tet(&tet, m, mode, &T[w], NULL, NULL, NULL);
                }
            }
    return 0;
}

/* Where the method's hard places are (used to aim the windows of the full-size parity tests):
 *   out[0..3]  = (i, j, k, t) of the tet with the largest cell range (ties: the first)
 *   out[4..6]  = its lo cell;  out[7] = its number of cells
 *   out[8..11] = (i, j, k, t) of the thinnest tet: smallest |det| / (product of the AABB edge
 *                lengths in cells), among non-degenerate tets whose range has >= min_cells cells
 *   out[12..14] = its lo cell; thin_out = that ratio                                          */
int psdo_extreme_tets(const void *pos, int dtype, int stride, int N, double L, int G,
                      int64_t min_cells, int64_t *out, double *thin_out) {
    if (N < 2 || G < 1) return 1;
    particles_t p = {pos, dtype, stride, N, L};
    const REAL scale = (REAL)G / (REAL)L;
    int64_t best_n = -1, bi[4] = {0, 0, 0, 0}, blo[3] = {0, 0, 0};
    double best_thin = 1e300;
    int64_t ti[4] = {0, 0, 0, 0}, tlo[3] = {0, 0, 0};
    for (int i = 0; i < N; ++i) {
        int64_t r_n = -1, r_i[4] = {0, 0, 0, 0}, r_lo[3] = {0, 0, 0};
        double r_thin = 1e300;
        int64_t s_i[4] = {0, 0, 0, 0}, s_lo[3] = {0, 0, 0};
#pragma omp parallel
        {
            int64_t m_n = -1, m_i[4] = {0, 0, 0, 0}, m_lo[3] = {0, 0, 0};
            double m_thin = 1e300;
            int64_t q_i[4] = {0, 0, 0, 0}, q_lo[3] = {0, 0, 0};
#pragma omp for schedule(static)
            for (int j = 0; j < N; ++j)
                for (int k = 0; k < N; ++k) {
                    REAL P[8][3];
                    cell_corners(&p, i, j, k, P);
                    for (int t = 0; t < 6; ++t) {
                        tet_t tet;
                        make_tet(P, t, scale, &tet);
                        int64_t n = 1;
                        double box = 1.0;
                        for (int x = 0; x < 3; ++x) {
                            n *= tet.hi[x] - tet.lo[x] + 1;
                            REAL mn = tet.g[0][x], mx = tet.g[0][x];
                            for (int v = 1; v < 4; ++v) {
                                if (tet.g[v][x] < mn) mn = tet.g[v][x];
                                if (tet.g[v][x] > mx) mx = tet.g[v][x];
                            }
                            box *= (double)(mx - mn);
                        }
                        if (n > m_n) {
                            m_n = n; m_i[0] = i; m_i[1] = j; m_i[2] = k; m_i[3] = t;
                            for (int x = 0; x < 3; ++x) m_lo[x] = tet.lo[x];
                        }
                        double d = (double)(tet.det < 0 ? -tet.det : tet.det);
                        if (n >= min_cells && d > 0 && box > 0 && d / box < m_thin) {
                            m_thin = d / box; q_i[0] = i; q_i[1] = j; q_i[2] = k; q_i[3] = t;
                            for (int x = 0; x < 3; ++x) q_lo[x] = tet.lo[x];
                        }
                    }
                }
#pragma omp critical
            {
                /* ties by (j,k,t) order: keep the smallest flat index */
                int64_t key_m = (m_i[1] * N + m_i[2]) * 6 + m_i[3], key_r = (r_i[1] * N + r_i[2]) * 6 + r_i[3];
                if (m_n > r_n || (m_n == r_n && m_n >= 0 && key_m < key_r)) {
                    r_n = m_n;
                    for (int x = 0; x < 4; ++x) r_i[x] = m_i[x];
                    for (int x = 0; x < 3; ++x) r_lo[x] = m_lo[x];
                }
                if (m_thin < r_thin) {
                    r_thin = m_thin;
                    for (int x = 0; x < 4; ++x) s_i[x] = q_i[x];
                    for (int x = 0; x < 3; ++x) s_lo[x] = q_lo[x];
                }
            }
        }
        if (r_n > best_n) {
            best_n = r_n;
            for (int x = 0; x < 4; ++x) bi[x] = r_i[x];
            for (int x = 0; x < 3; ++x) blo[x] = r_lo[x];
        }
        if (r_thin < best_thin) {
            best_thin = r_thin;
            for (int x = 0; x < 4; ++x) ti[x] = s_i[x];
            for (int x = 0; x < 3; ++x) tlo[x] = s_lo[x];
        }
    }
    for (int x = 0; x < 4; ++x) { out[x] = bi[x]; out[8 + x] = ti[x]; }
    for (int x = 0; x < 3; ++x) { out[4 + x] = blo[x]; out[12 + x] = tlo[x]; }
    out[7] = best_n;
    if (thin_out) *thin_out = best_thin;
    return 0;
}

/* ---- single-tet entry points used by the pins -------------------------------- */

/* vol(T n [lo, lo+h]^3) for an arbitrary tet given in any units (12 doubles, v-major). */
double psdo_tet_box_volume(const double *verts, const double *lo, double h) {
    REAL t[4][3];
    for (int v = 0; v < 4; ++v)
        for (int x = 0; x < 3; ++x) t[v][x] = ((REAL)verts[3 * v + x] - (REAL)lo[x]) / (REAL)h;
    return (double)(split_clip(t, 0) * (REAL)h * (REAL)h * (REAL)h);
}

/* vol(T n {lo <= x <= hi per axis}) for a general box: scale each axis to the unit cell. */
double psdo_tet_aabox_volume(const double *verts, const double *lo, const double *hi) {
    REAL t[4][3];
    REAL jac = 1;
    for (int x = 0; x < 3; ++x) {
        REAL e = (REAL)hi[x] - (REAL)lo[x];
        jac *= e;
        for (int v = 0; v < 4; ++v) t[v][x] = ((REAL)verts[3 * v + x] - (REAL)lo[x]) / e;
    }
    return (double)(split_clip(t, 0) * jac);
}

/* Overlap volumes (cell units) of one tet given in GRID units with every cell of the box
 * lo[x] <= c < lo[x]+n[x]; out is n0*n1*n2.  Returns |V| (cell units) via *vol_out.     */
int psdo_tet_deposit_box(const double *verts, const int64_t *lo, const int64_t *n, double *out,
                         double *vol_out) {
    REAL g[4][3];
    for (int v = 0; v < 4; ++v)
        for (int x = 0; x < 3; ++x) g[v][x] = (REAL)verts[3 * v + x];
    for (int64_t a = 0; a < n[0]; ++a)
        for (int64_t b = 0; b < n[1]; ++b)
            for (int64_t c = 0; c < n[2]; ++c) {
                int64_t cc[3] = {lo[0] + a, lo[1] + b, lo[2] + c};
                out[(a * n[1] + b) * n[2] + c] = (double)tet_cell_volume(g, cc);
            }
    if (vol_out) {
        DETREAL d = det3(g);
        *vol_out = (double)((d < 0 ? -d : d) / (DETREAL)6);
    }
    return 0;
}

/* The 4 unwrapped vertices (box units) of tet t of Lagrangian cell (i,j,k), its signed
 * determinant in GRID units (G cells per L) and its cell range. */
int psdo_build_tet(const void *pos, int dtype, int stride, int N, double L, int G, int i, int j,
                   int k, int t, double *verts_out, double *det_out, int64_t *lohi_out) {
    if (t < 0 || t > 5) return 1;
    particles_t p = {pos, dtype, stride, N, L};
    REAL P[8][3];
    cell_corners(&p, i, j, k, P);
    tet_t tet;
    make_tet(P, t, (REAL)G / (REAL)L, &tet);
    for (int v = 0; v < 4; ++v)
        for (int x = 0; x < 3; ++x) verts_out[3 * v + x] = (double)P[KUHN[t][v]][x];
    if (det_out) *det_out = (double)tet.det;
    if (lohi_out)
        for (int x = 0; x < 3; ++x) { lohi_out[x] = tet.lo[x]; lohi_out[3 + x] = tet.hi[x]; }
    return 0;
}

void psdo_kuhn_table(int *out24) {
    for (int t = 0; t < 6; ++t)
        for (int v = 0; v < 4; ++v) out24[4 * t + v] = KUHN[t][v];
}

/* ---- O6: patches (Q13).  A patch is {level, ox, oy, oz}: it
 * covers cells [o*P, o*P+P) of the level grid G_l = base_G * 2^level.  Every listed
 * patch receives the full deposit of every tet overlapping it.                        */
typedef struct { int32_t level, ox, oy, oz; } psdo_patch;

/* per_patch (optional): [q*2+0] candidate cells, [q*2+1] cells with non-zero overlap of patch q
 * (counters only; the arithmetic is that of psdo_deposit_patches). */
int psdo_deposit_patches_stats(const void *pos, int dtype, int stride, int N, double L, double M,
                               int base_G, int P, const psdo_patch *patches, int64_t n_patch,
                               double *mass, int mode, int64_t *per_patch) {
    if (N < 2 || base_G < 1 || P < 1 || base_G % P) return 1;
    memset(mass, 0, sizeof(double) * (size_t)(n_patch * P * P * P));
    int rc = 0;
    for (int64_t q = 0; q < n_patch; ++q) {
        int64_t G = (int64_t)base_G << patches[q].level;
        int64_t wlo[3] = {(int64_t)patches[q].ox * P, (int64_t)patches[q].oy * P,
                          (int64_t)patches[q].oz * P};
        int64_t wn[3] = {P, P, P};
        target_t T = {G, mass + q * (int64_t)P * P * P, 1, {wlo[0], wlo[1], wlo[2]},
                      {wn[0], wn[1], wn[2]}};
        int64_t st[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        rc |= deposit_common(pos, dtype, stride, N, L, M, (int)G, &T, mode, st);
        if (per_patch) { per_patch[2 * q] = st[1]; per_patch[2 * q + 1] = st[2]; }
    }
    return rc;
}

int psdo_deposit_patches(const void *pos, int dtype, int stride, int N, double L, double M,
                         int base_G, int P, const psdo_patch *patches, int64_t n_patch,
                         double *mass, int mode) {
    return psdo_deposit_patches_stats(pos, dtype, stride, N, L, M, base_G, P, patches, n_patch, mass,
                                      mode, NULL);
}

/* counts[l] is a dense (base_G/P * 2^l)^3 array: number of tets whose cell range on the
 * level-l grid meets patch position (px,py,pz) (each position once per tet).  PAPER.md:66. */
int psdo_patch_counts(const void *pos, int dtype, int stride, int N, double L, int base_G, int P,
                      int level, uint64_t *counts) {
    if (N < 2 || base_G % P) return 1;
    particles_t p = {pos, dtype, stride, N, L};
    const int64_t G = (int64_t)base_G << level;
    const int64_t np = G / P;
    const REAL scale = (REAL)G / (REAL)L;
    memset(counts, 0, sizeof(uint64_t) * (size_t)(np * np * np));
    unsigned char *seen[3];
    for (int x = 0; x < 3; ++x) seen[x] = (unsigned char *)malloc((size_t)np);
    for (int i = 0; i < N; ++i)
        for (int j = 0; j < N; ++j)
            for (int k = 0; k < N; ++k) {
                REAL Pc[8][3];
                cell_corners(&p, i, j, k, Pc);
                for (int t = 0; t < 6; ++t) {
                    tet_t tet;
                    make_tet(Pc, t, scale, &tet);
                    for (int x = 0; x < 3; ++x) {
                        memset(seen[x], 0, (size_t)np);
                        for (int64_t c = tet.lo[x]; c <= tet.hi[x]; ++c) seen[x][wrap(c, G) / P] = 1;
                    }
                    for (int64_t a = 0; a < np; ++a) {
                        if (!seen[0][a]) continue;
                        for (int64_t b = 0; b < np; ++b) {
                            if (!seen[1][b]) continue;
                            for (int64_t c = 0; c < np; ++c)
                                if (seen[2][c]) counts[(a * np + b) * np + c]++;
                        }
                    }
                }
            }
    for (int x = 0; x < 3; ++x) free(seen[x]);
    return 0;
}

/* O7.  counts[] is the dense (base_G/P * 2^level)^3 array of candidate patch
 * positions; each receives, from every sub-block of B^3 Lagrangian cells (the last one per
 * axis may be smaller), T_b * vol(AABB n patch) / vol(AABB) in units of 2^-20 tets, rounded
 * to the nearest integer per (sub-block, patch) so that the sum does not depend on the order
 * (T_b = 6 x cells of the sub-block; the AABB spans the sub-block's particles including the
 * layer shared with the next sub-block, unwrapped to the minimum image of its first
 * particle).  All arithmetic in double, one rounding per operation. */
int psdo_subblock_counts(const void *pos, int dtype, int stride, int N, double L, int base_G, int P,
                         int level, int B, uint64_t *counts) {
    if (N < 2 || base_G % P || B < 1) return 1;
    particles_t p = {pos, dtype, stride, N, L};
    const int64_t G = (int64_t)base_G << level;
    const int64_t np = G / P;
    const double scale = (double)G / L;
    const double Pc = (double)P;
    memset(counts, 0, sizeof(uint64_t) * (size_t)(np * np * np));
    const int nb = (N + B - 1) / B;
    for (int bi = 0; bi < nb; ++bi)
        for (int bj = 0; bj < nb; ++bj)
            for (int bk = 0; bk < nb; ++bk) {
                int o[3] = {bi * B, bj * B, bk * B}, n[3];
                for (int x = 0; x < 3; ++x) n[x] = (o[x] + B <= N) ? B : N - o[x];
                double ref[3], lo[3], hi[3];
                int64_t ridx = ((int64_t)o[0] * N + o[1]) * N + o[2];
                for (int c = 0; c < 3; ++c) lo[c] = hi[c] = ref[c] = (double)load_coord(&p, ridx, c);
                for (int a = 0; a <= n[0]; ++a)
                    for (int b = 0; b <= n[1]; ++b)
                        for (int cc = 0; cc <= n[2]; ++cc) {
                            int64_t idx = ((int64_t)((o[0] + a) % N) * N + (o[1] + b) % N) * N + (o[2] + cc) % N;
                            for (int c = 0; c < 3; ++c) {
                                double xv = (double)load_coord(&p, idx, c);
                                double d = xv - ref[c];
                                double q = d / L;
                                double r = rint(q);
                                double sft = L * r;
                                xv = xv - sft;
                                if (xv < lo[c]) lo[c] = xv;
                                if (xv > hi[c]) hi[c] = xv;
                            }
                        }
                const double Tfix = (double)(6 * (int64_t)n[0] * n[1] * n[2]) * 1048576.0;
                int64_t first[3], cnt[3];
                double frac[3][64];
                int too_many = 0;
                for (int x = 0; x < 3; ++x) {
                    double glo = lo[x] * scale, ghi = hi[x] * scale;
                    double ext = ghi - glo;
                    first[x] = (int64_t)floor(glo / Pc);
                    int64_t last = (int64_t)floor(ghi / Pc);
                    cnt[x] = last - first[x] + 1;
                    if (cnt[x] > 64) { too_many = 1; break; }
                    for (int64_t q = 0; q < cnt[x]; ++q) {
                        double a = (double)((first[x] + q) * P), b = (double)((first[x] + q + 1) * P);
                        if (glo > a) a = glo;
                        if (ghi < b) b = ghi;
                        double ov = b - a;
                        if (ov < 0.0) ov = 0.0;
                        frac[x][q] = ext > 0.0 ? ov / ext : 1.0;
                    }
                }
                if (too_many) return 2;
                for (int64_t a = 0; a < cnt[0]; ++a)
                    for (int64_t b = 0; b < cnt[1]; ++b)
                        for (int64_t c = 0; c < cnt[2]; ++c) {
                            double f = frac[0][a] * frac[1][b];
                            f = f * frac[2][c];
                            double e = Tfix * f;
                            e = e + 0.5;
                            uint64_t est = (uint64_t)floor(e);
                            counts[(wrap(first[0] + a, np) * np + wrap(first[1] + b, np)) * np +
                                   wrap(first[2] + c, np)] += est;
                        }
            }
    return 0;
}

int psdo_is_gold(void) {
#ifdef PSDO_GOLD
    return 1;
#else
    return 0;
#endif
}

int psdo_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

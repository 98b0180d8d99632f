// psd_geom.cuh -- device-side geometry of the phase-space-element deposit (sm_100a).
//
// What is computed (PAPER.md = /root/reference/PAPER.md, arXiv:1612.09491):
//   PAPER.md:39-45   tets generated on the fly from the Lagrangian lattice (6 per cell)
//   PAPER.md:137     mass += m * vol(T n C) / |vol(T)|
//   PAPER.md:155-161 exact tet-cube intersection by axis-aligned plane clipping
//
// How (differs from the paper's K80 design):
// the tet is kept as a boundary polytope (its 4 oriented faces).  The unit of work is a
// FACE JOB: one face triangle against one COLUMN of cells (a unit square in two axes, running
// along the third, "chord" axis u).  The triangle is clipped by the (at most 4) axis-aligned walls
// of the column it crosses -- a convex polygon meets a line on exactly two edges, so a clip is two
// interpolations and a re-packed vertex order -- giving a convex polygon Q, on which u is linear.
// With
//     R_F(a) = signed integral over Q n {u >= a} of (u - a) dv dw
// the divergence theorem (flux of (u-a,0,0)) gives, summed over the 4 faces,
//     R(a) = vol(T n column n {u >= a}),
// so the cell [a,a+1] receives R(a) - R(a+1): the cell's own faces never need a cap polygon
// (column walls have zero u-flux and the cap u = a has u-a = 0), and every face adds its own
// share to the cell independently of the other faces.  R_F(a) = M1 - a A below Q, 0 above it, and
// for a plane that cuts Q the part above the plane is fanned from its first crossing with the
// plane (plane_integral6): a sum of same-signed terms, a few flops per vertex, not another stored
// clip.  All interpolation is between points on opposite sides of a plane (convex combinations),
// every ratio used is in [0,1], coordinates are local to the tile/column, arithmetic is fp64.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace psd {

constexpr int TILE = 8;            // tile edge in cells (BASELINE north_star: 8^3-cell tiles)
constexpr int TILE_CELLS = 512;
constexpr int POLY_CAP = 7;        // triangle + 4 column planes -> <= 7 vertices, slots 0..6

// Kuhn / Freudenthal split: every tet is (corner 0, a, b, corner 7); corner index
// bit0 = +x, bit1 = +y, bit2 = +z.  Own copy (the oracle has its own).
__device__ __constant__ int c_kuhn_mid[6][2] = {{1, 3}, {5, 1}, {3, 2}, {2, 6}, {4, 5}, {6, 4}};

struct Particles {
    const void* pos;
    int dtype;   // 0 f32, 1 f64
    int stride;  // 3 or 4
    int N;
    double L;
    double inv_L;  // 1 / L when L is a power of two (then x * inv_L == x / L exactly), else 0
};

__device__ __forceinline__ void load_pos(const Particles& p, int64_t idx, double out[3]) {
    if (p.dtype == 0) {
        if (p.stride == 4) {
            float4 v = __ldg(reinterpret_cast<const float4*>(p.pos) + idx);
            out[0] = (double)v.x; out[1] = (double)v.y; out[2] = (double)v.z;
        } else {
            const float* f = reinterpret_cast<const float*>(p.pos) + idx * 3;
            out[0] = (double)__ldg(f); out[1] = (double)__ldg(f + 1); out[2] = (double)__ldg(f + 2);
        }
    } else {
        const double* d = reinterpret_cast<const double*>(p.pos) + idx * p.stride;
        out[0] = __ldg(d); out[1] = __ldg(d + 1); out[2] = __ldg(d + 2);
    }
}

// minimum image of `ref` (PAPER.md silent; Q3/Q4).  Individually rounded IEEE ops
// (no FMA contraction) so the integer cell ranges match the oracle bit for bit.
__device__ __forceinline__ double unwrap1(double x, double ref, double L, double inv_L) {
    double d = __dsub_rn(x, ref);
    // d / L, correctly rounded as in the oracle; when L is a power of two the product with the
    // (exact) reciprocal is the same number and spares the division's long instruction sequence
    double q = inv_L != 0.0 ? __dmul_rn(d, inv_L) : __ddiv_rn(d, L);
    double r = rint(q);
    double s = __dmul_rn(L, r);
    return __dsub_rn(x, s);
}

__device__ __forceinline__ int64_t corner_index(int i, int j, int k, int b, int N) {
    int ii = i + (b & 1), jj = j + ((b >> 1) & 1), kk = k + ((b >> 2) & 1);
    ii = ii == N ? 0 : ii; jj = jj == N ? 0 : jj; kk = kk == N ? 0 : kk;
    return ((int64_t)ii * N + jj) * N + kk;
}

// ---- error-free transforms for the tet determinant (denominator of the mass weight) ----
__device__ __forceinline__ void two_sum(double a, double b, double& s, double& e) {
    s = __dadd_rn(a, b);
    double bb = __dsub_rn(s, a);
    e = __dadd_rn(__dsub_rn(a, __dsub_rn(s, bb)), __dsub_rn(b, bb));
}
__device__ __forceinline__ void two_prod(double a, double b, double& p, double& e) {
    p = __dmul_rn(a, b);
    e = __fma_rn(a, b, -p);
}
// (h,l) = a*b - c*d to nearly twice working precision
__device__ __forceinline__ void dd_minor(double a, double b, double c, double d, double& h, double& l) {
    double p1, e1, p2, e2, s, t;
    two_prod(a, b, p1, e1);
    two_prod(c, d, p2, e2);
    two_sum(p1, -p2, s, t);
    l = __dadd_rn(t, __dsub_rn(e1, e2));
    h = s;
}
// x * (h,l) as (ph, pl)
__device__ __forceinline__ void dd_scale(double x, double h, double l, double& ph, double& pl) {
    double e;
    two_prod(x, h, ph, e);
    pl = __fma_rn(x, l, e);
}
__device__ __forceinline__ double det3_plain(const double a[3], const double b[3], const double c[3]) {
    return a[0] * (b[1] * c[2] - b[2] * c[1]) - a[1] * (b[0] * c[2] - b[2] * c[0]) +
           a[2] * (b[0] * c[1] - b[1] * c[0]);
}
// det(v1-v0, v2-v0, v3-v0), compensated: edge differences as (hi,lo) pairs, the leading
// determinant in double-double, first-order corrections for the lo parts.
__device__ __forceinline__ double tet_det(const double g[4][3]) {
    double ah[3], al[3], bh[3], bl[3], ch[3], cl[3];
#pragma unroll
    for (int x = 0; x < 3; ++x) {
        two_sum(g[1][x], -g[0][x], ah[x], al[x]);
        two_sum(g[2][x], -g[0][x], bh[x], bl[x]);
        two_sum(g[3][x], -g[0][x], ch[x], cl[x]);
    }
    double m0h, m0l, m1h, m1l, m2h, m2l;
    dd_minor(bh[1], ch[2], bh[2], ch[1], m0h, m0l);
    dd_minor(bh[0], ch[2], bh[2], ch[0], m1h, m1l);
    dd_minor(bh[0], ch[1], bh[1], ch[0], m2h, m2l);
    double t0h, t0l, t1h, t1l, t2h, t2l;
    dd_scale(ah[0], m0h, m0l, t0h, t0l);
    dd_scale(-ah[1], m1h, m1l, t1h, t1l);
    dd_scale(ah[2], m2h, m2l, t2h, t2l);
    double s, e1, e2;
    two_sum(t0h, t1h, s, e1);
    two_sum(s, t2h, s, e2);
    double lo = __dadd_rn(__dadd_rn(e1, e2), __dadd_rn(__dadd_rn(t0l, t1l), t2l));
    lo += det3_plain(al, bh, ch) + det3_plain(ah, bl, ch) + det3_plain(ah, bh, cl);
    return s + lo;
}

// Sign of the determinant only (census statistics: inverted / degenerate counts): the plain
// determinant of the rounded edge vectors when it clears a bound on its own rounding error
// (a few ulp of the product of the edges' 1-norms, taken 400x wider here), else the compensated one.
__device__ __forceinline__ double tet_det_sign(const double g[4][3]) {
    double a[3], b[3], c[3];
#pragma unroll
    for (int x = 0; x < 3; ++x) { a[x] = g[1][x] - g[0][x]; b[x] = g[2][x] - g[0][x]; c[x] = g[3][x] - g[0][x]; }
    const double d = det3_plain(a, b, c);
    const double bound = (fabs(a[0]) + fabs(a[1]) + fabs(a[2])) * (fabs(b[0]) + fabs(b[1]) + fabs(b[2])) *
                         (fabs(c[0]) + fabs(c[1]) + fabs(c[2]));
    return fabs(d) > 1e-13 * bound ? d : tet_det(g);
}

__device__ __forceinline__ int floor_div(int a, int b) {  // b > 0
    int q = a / b, r = a % b;
    return (r != 0 && r < 0) ? q - 1 : q;
}
__device__ __forceinline__ int wrap_mod(int a, int b) {  // b > 0
    int r = a % b;
    return r < 0 ? r + b : r;
}
__device__ __forceinline__ int bit_width_u64(unsigned long long v) { return 64 - __clzll((long long)v); }

// One tetrahedron on a grid of G cells per side: vertices in grid units (unwrapped), integer
// cell range, signed determinant (= 6 * signed volume, grid units).
struct Tet {
    double g[4][3];
    int lo[3], hi[3];
    double det;
};

// Build from the 4 box-unit vertices already unwrapped.
__device__ __forceinline__ void finish_tet(const double P[4][3], double scale, Tet& t) {
#pragma unroll
    for (int v = 0; v < 4; ++v)
#pragma unroll
        for (int x = 0; x < 3; ++x) t.g[v][x] = __dmul_rn(P[v][x], scale);
#pragma unroll
    for (int x = 0; x < 3; ++x) {
        double mn = fmin(fmin(t.g[0][x], t.g[1][x]), fmin(t.g[2][x], t.g[3][x]));
        double mx = fmax(fmax(t.g[0][x], t.g[1][x]), fmax(t.g[2][x], t.g[3][x]));
        t.lo[x] = __double2int_rd(mn);
        t.hi[x] = __double2int_rd(mx);
    }
}

// Load + unwrap the 4 vertices of tet `t6` (0..5) of Lagrangian cell `cell` (box units).
__device__ __forceinline__ void load_tet_vertices(const Particles& p, int64_t cell, int t6,
                                                  double P[4][3]) {
    const int N = p.N;
    int k = (int)(cell % N), j = (int)((cell / N) % N), i = (int)(cell / ((int64_t)N * N));
    int ca = c_kuhn_mid[t6][0], cb = c_kuhn_mid[t6][1];
    load_pos(p, corner_index(i, j, k, 0, N), P[0]);
    load_pos(p, corner_index(i, j, k, ca, N), P[1]);
    load_pos(p, corner_index(i, j, k, cb, N), P[2]);
    load_pos(p, corner_index(i, j, k, 7, N), P[3]);
#pragma unroll
    for (int v = 1; v < 4; ++v)
#pragma unroll
        for (int x = 0; x < 3; ++x) P[v][x] = unwrap1(P[v][x], P[0][x], p.L, p.inv_L);
}

// 1/x to about 1 ulp for a normal, non-zero x, without the IEEE division's special-case path:
// hardware seed (MUFU.RCP64H) and two Newton steps.  The clip ratios do not need correct rounding.
__device__ __forceinline__ double fast_rcp(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    r = fma(fma(-x, r, 1.0), r, r);
    r = fma(fma(-x, r, 1.0), r, r);
    return r;
}

// ------------------------------------------------------------------ polygon buffer
// One lane's polygon: POLY_CAP vertices x (u,v,w), element stride S doubles
// (S = 32: warp-interleaved shared memory, bank-conflict free for any index; S = 1: local).
template <int S>
struct PolyBuf {
    double* p;
    __host__ __device__ __forceinline__ double& at(int i, int c) { return p[(3 * i + c) * S]; }
};


// A convex polygon as a CYCLIC ORDER over storage slots: nibble i of `order` is the slot (0..6)
// holding vertex i; vertices never move, a clip only writes its two new points and re-packs the
// order word.  Slots 0..2 hold the face triangle; each clip allocates at most one fresh slot
// (`fresh`), so 3 + 4 walls = 7 slots suffice (POLY_CAP).
struct PolyRef {
    unsigned order;
    unsigned oc;  // nibble i = outcode of vertex i: bit k set = inside wall k (0: v>=0, 1: v<=1, 2: w>=0, 3: w<=1)
    int n;
    int fresh;
};

// bit k of every nibble of x (7 nibbles) gathered into bits 0..6
__device__ __forceinline__ unsigned gather_nibble_bit(unsigned x, int k) {
    unsigned y = (x >> k) & 0x01111111u;
    y = (y | (y >> 3)) & 0x03030303u;
    y = (y | (y >> 6)) & 0x000f000fu;
    return (y | (y >> 12)) & 0x7fu;
}

__host__ __device__ __forceinline__ int slot_of(unsigned order, int i) { return (order >> (4 * i)) & 15; }
__device__ __forceinline__ unsigned nib_mask(int n) { return n >= 8 ? 0xffffffffu : ((1u << (4 * n)) - 1u); }

// The two edges where a convex polygon with inside-bits `mask` (bit i: vertex i inside, neither
// empty nor full) crosses a line: i_out = first outside vertex after an inside one, i_in = first
// inside vertex after an outside one (cyclic).
__device__ __forceinline__ void crossing_edges(unsigned mask, int n, int& i_out, int& i_in) {
    const unsigned full = (1u << n) - 1u;
    const unsigned prev = ((mask << 1) | (mask >> (n - 1))) & full;  // bit i = inside(i-1)
    i_out = __ffs(prev & ~mask) - 1;
    i_in = __ffs(~prev & mask & full) - 1;
}

// Clip the polygon against one wall of the column: wall 0: v >= 0, 1: v <= 1, 2: w >= 0,
// 3: w <= 1 (a runtime value, so lanes clipping different walls run the same instructions).
// Vertices exactly on the wall are inside; a convex polygon crosses the wall on exactly two edges,
// each crossing is interpolated from its inside endpoint (ratio in [0,1]) and, with SNAP, put exactly on the wall.
template <int S, bool SNAP>
__device__ __forceinline__ void clip_wall(PolyBuf<S> q, PolyRef& r, int wall) {
    const int ax = 1 + (wall >> 1);
    const bool up = wall & 1;
    const unsigned mask = gather_nibble_bit(r.oc, wall);
    const unsigned full = (1u << r.n) - 1u;
    if (mask == full) return;
    if (mask == 0) { r.n = 0; return; }
    int i_out, i_in;
    crossing_edges(mask, r.n, i_out, i_in);
    const int sa = slot_of(r.order, i_out ? i_out - 1 : r.n - 1), sb = slot_of(r.order, i_out);
    const int sc = slot_of(r.order, i_in ? i_in - 1 : r.n - 1), se = slot_of(r.order, i_in);
    // signed distance to the wall: d = sgn * x + wallpos (inside: d >= 0)
    const double sgn = up ? -1.0 : 1.0, wallpos = up ? 1.0 : 0.0;
    const double da = fma(sgn, q.at(sa, ax), wallpos), db = fma(sgn, q.at(sb, ax), wallpos);
    const double de = fma(sgn, q.at(se, ax), wallpos), dc = fma(sgn, q.at(sc, ax), wallpos);
    const double t1 = da * fast_rcp(da - db);  // leaving crossing: inside a -> outside b
    const double t2 = de * fast_rcp(de - dc);  // entering crossing: inside e -> outside c
    double xo[3], xi[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double a = q.at(sa, c), e = q.at(se, c);
        xo[c] = fma(t1, q.at(sb, c) - a, a);
        xi[c] = fma(t2, q.at(sc, c) - e, e);
    }
    // put the new points exactly on the wall where that is free (compile-time wall id); with a
    // runtime wall id it costs 8 selects and changes nothing: the new points' outcodes for this
    // wall are set, not computed, and an offset of one rounding error is below the clip's own
    if (SNAP) { if (ax == 1) { xo[1] = wallpos; xi[1] = wallpos; } else { xo[2] = wallpos; xi[2] = wallpos; } }
    // new points go to the slots of the first and last removed vertex (already read); if only one
    // vertex was removed the second point takes a fresh slot
    const int s_out = sb;
    int s_in = sc;
    if (sc == sb) s_in = r.fresh++;
#pragma unroll
    for (int c = 0; c < 3; ++c) { q.at(s_out, c) = xo[c]; q.at(s_in, c) = xi[c]; }
    // order: X_in, the inside run (starting at i_in), X_out
    const int m = __popc(mask);
    const unsigned rot = i_in ? ((r.order >> (4 * i_in)) | (r.order << (4 * (r.n - i_in)))) : r.order;
    const unsigned roc = i_in ? ((r.oc >> (4 * i_in)) | (r.oc << (4 * (r.n - i_in)))) : r.oc;
    // outcodes of the new points: on this wall and inside the opposite one; the other axis by compare
    const unsigned own = ax == 1 ? 3u : 12u;
    const double yo = ax == 1 ? xo[2] : xo[1], yi = ax == 1 ? xi[2] : xi[1];
    const int sh = ax == 1 ? 2 : 0;
    const unsigned oc_out = own | ((unsigned)(yo >= 0.0) | (unsigned)(yo <= 1.0) << 1) << sh;
    const unsigned oc_in = own | ((unsigned)(yi >= 0.0) | (unsigned)(yi <= 1.0) << 1) << sh;
    r.order = (unsigned)s_in | ((rot & nib_mask(m)) << 4) | ((unsigned)s_out << (4 * (m + 1)));
    r.oc = oc_in | ((roc & nib_mask(m)) << 4) | (oc_out << (4 * (m + 1)));
    r.n = m + 2;
}

// R(a) = integral over Q n {u >= a} of (u - a) dv dw for a plane strictly between the polygon's
// lowest and highest vertex: Q is cut by the line u = a (two crossings X_in, X_out with u - a = 0,
// not stored), and the kept part [X_in, inside run, X_out] is fanned from X_in.  Every fan triangle
// lies inside Q and every height is >= 0: a sum of same-signed terms, no cancellation.
// Returns 6 R (signed like the polygon's orientation).
template <int S>
__device__ __forceinline__ double plane_integral6_mask(PolyBuf<S> q, unsigned order, int n, double a, unsigned mask);

template <int S>
__device__ __forceinline__ double plane_integral6(PolyBuf<S> q, unsigned order, int n, double a) {
    unsigned mask = 0;
#pragma unroll
    for (int i = 0; i < POLY_CAP; ++i) {
        if (i >= n) break;
        mask |= (unsigned)(q.at(slot_of(order, i), 0) >= a) << i;
    }
    return plane_integral6_mask<S>(q, order, n, a, mask);
}

// Vertex i is at or above the lattice plane a  <=>  floor(u_i) >= a: with the floors of the
// polygon's vertex heights packed one nibble each (clamped to 0..8) the inside mask of a plane
// 1..8 is one add and a bit gather, no loads; plane 0 takes the mask of the vertices below 0.
__device__ __forceinline__ unsigned plane_mask_from_floors(unsigned floors, unsigned below0, int n, int a) {
    const unsigned full = (1u << n) - 1u;
    if (a == 0) return full & ~below0;  // plane 0: every vertex that is not below the tile
    return gather_nibble_bit(floors + (unsigned)(8 - a) * 0x01111111u, 3) & full;
}

// the integral proper, inside-mask given (bit i: vertex i has u >= a)
template <int S>
__device__ __forceinline__ double plane_integral6_mask(PolyBuf<S> q, unsigned order, int n, double a, unsigned mask) {
    const unsigned full = (1u << n) - 1u;
    if (mask == 0 || mask == full) return 0.0;  // not a cutting plane (caller excludes this)
    int i_out, i_in;
    crossing_edges(mask, n, i_out, i_in);
    const int sa = slot_of(order, i_out ? i_out - 1 : n - 1), sb = slot_of(order, i_out);
    const int sc = slot_of(order, i_in ? i_in - 1 : n - 1);
    double x0v, x0w, xov, xow;
    {
        const double ha = q.at(sa, 0) - a, hb = q.at(sb, 0) - a;
        const double t = ha * fast_rcp(ha - hb);
        const double av = q.at(sa, 1), aw = q.at(sa, 2);
        xov = fma(t, q.at(sb, 1) - av, av); xow = fma(t, q.at(sb, 2) - aw, aw);
    }
    const unsigned rot = i_in ? ((order >> (4 * i_in)) | (order << (4 * (n - i_in)))) : order;
    const int m = __popc(mask);
    double pv, pw, ph;  // first inside vertex, relative to X_in
    {
        const int se = rot & 15;
        const double he = q.at(se, 0) - a, hc = q.at(sc, 0) - a;
        const double t = he * fast_rcp(he - hc);
        const double ev = q.at(se, 1), ew = q.at(se, 2);
        x0v = fma(t, q.at(sc, 1) - ev, ev); x0w = fma(t, q.at(sc, 2) - ew, ew);
        pv = ev - x0v; pw = ew - x0w; ph = he;
    }
    double sum = 0.0;
#pragma unroll
    for (int j = 1; j < POLY_CAP; ++j) {  // the inside vertices after the first
        if (j >= m) break;
        const int s = (rot >> (4 * j)) & 15;
        const double cv = q.at(s, 1) - x0v, cw = q.at(s, 2) - x0w, ch = q.at(s, 0) - a;
        sum = fma(pv * cw - pw * cv, ph + ch, sum);
        pv = cv; pw = cw; ph = ch;
    }
    sum = fma(pv * (xow - x0w) - pw * (xov - x0v), ph, sum);  // last triangle: up to X_out (height 0)
    return sum;
}

struct JobCounters {
    unsigned int jobs, face_clips, plane_evals, cells, general;
};

// faces of tet (0,1,2,3) with outward orientation when det > 0: (1,2,3) (0,3,2) (0,1,3) (0,2,1)
// packed 2 bits per vertex index, 6 bits per face.
constexpr unsigned FACE_TABLE = (1u | 2u << 2 | 3u << 4) | (0u | 3u << 2 | 2u << 4) << 6 |
                                (0u | 1u << 2 | 3u << 4) << 12 | (0u | 2u << 2 | 1u << 4) << 18;

// Result of clipping one face triangle to one column (Q = triangle n column).
struct FaceClip {
    unsigned order;
    int n;            // 0: empty
    double A, M1;     // signed projected area of Q, first moment integral of u over Q
    int ifl, ice;     // floor of the lowest, ceil of the highest vertex height
    unsigned floors;  // nibble i = floor of vertex i's height, clamped to 0..8 (plane_mask_from_floors)
    unsigned below0;  // bit i = vertex i's height is below 0
};

// q holds the face triangle in slots 0..2: (u, v, w) with v, w relative to the column's lower
// corner (the column is the unit square [0,1]^2).
// tri_outcodes: outcodes of that triangle (nibble i = vertex i, see PolyRef::oc), their AND and OR.
template <int S>
__device__ __forceinline__ unsigned tri_outcodes(PolyBuf<S> q, unsigned& all_in, unsigned& any_in) {
    unsigned oc = 0;
    all_in = 15u; any_in = 0u;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const double v = q.at(i, 1), w = q.at(i, 2);
        const unsigned o = (unsigned)(v >= 0.0) | (unsigned)(v <= 1.0) << 1 | (unsigned)(w >= 0.0) << 2 |
                           (unsigned)(w <= 1.0) << 3;
        oc |= o << (4 * i);
        all_in &= o; any_in |= o;
    }
    return oc;
}

// Signed projected area A and first moment M1 = integral of u over the convex polygon
// (order, n), fanned from its vertex 0; floor / ceil of its lowest / highest vertex.
template <int S>
__device__ __forceinline__ FaceClip poly_area_moment(PolyBuf<S> q, unsigned order, int n) {
    FaceClip fc;
    fc.n = 0; fc.order = 0; fc.A = fc.M1 = 0.0; fc.ifl = fc.ice = 0; fc.floors = 0; fc.below0 = 0;
    if (n < 3) return fc;
    const int s0 = slot_of(order, 0), s1 = slot_of(order, 1);
    const double u0 = q.at(s0, 0), v0 = q.at(s0, 1), w0 = q.at(s0, 2);
    double lu = q.at(s1, 0), lv = q.at(s1, 1) - v0, lw = q.at(s1, 2) - w0;
    const int f0 = __double2int_rd(u0), f1 = __double2int_rd(lu);
    int ifl = min(f0, f1), ice = max(__double2int_ru(u0), __double2int_ru(lu));
    unsigned floors = (unsigned)min(max(f0, 0), 8) | (unsigned)min(max(f1, 0), 8) << 4;
    unsigned below0 = (unsigned)(f0 < 0) | (unsigned)(f1 < 0) << 1;
    double A2 = 0.0, M6 = 0.0;
#pragma unroll
    for (int i = 2; i < POLY_CAP; ++i) {
        if (i >= n) break;
        const int s = slot_of(order, i);
        const double cu = q.at(s, 0), cv = q.at(s, 1) - v0, cw = q.at(s, 2) - w0;
        const double cr = lv * cw - lw * cv;
        A2 += cr;
        M6 = fma(cr, u0 + lu + cu, M6);
        const int fi = __double2int_rd(cu);
        ifl = min(ifl, fi); ice = max(ice, __double2int_ru(cu));
        floors |= (unsigned)min(max(fi, 0), 8) << (4 * i);
        below0 |= (unsigned)(fi < 0) << i;
        lu = cu; lv = cv; lw = cw;
    }
    fc.order = order; fc.n = n; fc.floors = floors; fc.below0 = below0;
    fc.A = 0.5 * A2; fc.M1 = M6 * (1.0 / 6.0);
    fc.ifl = ifl; fc.ice = ice;
    return fc;
}

template <int S, bool WALLS_UNROLLED>
__device__ __forceinline__ FaceClip face_clip_oc(PolyBuf<S> q, unsigned oc, unsigned all_in, unsigned any_in);

template <int S, bool WALLS_UNROLLED = false>
__device__ __forceinline__ FaceClip face_clip(PolyBuf<S> q) {
    unsigned all_in, any_in;
    const unsigned oc = tri_outcodes<S>(q, all_in, any_in);
    return face_clip_oc<S, WALLS_UNROLLED>(q, oc, all_in, any_in);
}

// the clip proper, outcodes given (the pooled tile kernel computes them when it sorts the jobs)
template <int S, bool WALLS_UNROLLED>
__device__ __forceinline__ FaceClip face_clip_oc(PolyBuf<S> q, unsigned oc, unsigned all_in, unsigned any_in) {
    FaceClip fc;
    fc.n = 0; fc.order = 0; fc.A = fc.M1 = 0.0; fc.ifl = fc.ice = 0; fc.floors = 0; fc.below0 = 0;
    if (any_in != 15u) return fc;  // all three vertices outside one wall
    PolyRef r{0x210u, oc, 3, 3};
    unsigned pending = all_in ^ 15u;
    if (WALLS_UNROLLED) {
        // the 4 walls in turn with a compile-time wall id (axis, side and outcode bit folded):
        // pays in the thread-per-tet kernel, not in the tile kernel (code size, registers)
#pragma unroll
        for (int wall = 0; wall < 4; ++wall)
            if (((pending >> wall) & 1u) && r.n) clip_wall<S, true>(q, r, wall);
    } else {
        while (pending && r.n) {
            const int wall = __ffs(pending) - 1;
            pending &= pending - 1;
            clip_wall<S, false>(q, r, wall);
        }
    }
    return poly_area_moment<S>(q, r.order, r.n);
}

// Cells and planes of a clipped face over the run of cells c_lo..c_hi (cell c spans u in [c,c+1]).
// The face's signed share of cell c is D(c) = R(c) - R(c+1), R(a) = integral over Q n {u >= a} of
// (u - a) dv dw:  R(a) = M1 - a A for a <= umin, 0 for a >= umax, plane_integral6/6 in between.
//   trivial part   cells c_lo..t_hi:  A if c+1 <= umin, else M1 - c A (the cell holding umin)
//   cutting planes a_first..a_last (umin < a < umax): +R(a) to cell a (if <= c_hi), -R(a) to
//                  cell a-1 (if >= c_lo)
struct FaceRun {
    int t_hi;             // last cell of the trivial part (< c_lo: none)
    int a_first, a_last;  // cutting planes (a_last < a_first: none)
};
__device__ __forceinline__ FaceRun face_run(const FaceClip& fc, int c_lo, int c_hi) {
    FaceRun fr;
    fr.t_hi = c_lo - 1; fr.a_first = 0; fr.a_last = -1;
    if (fc.n < 3 || fc.ice <= c_lo) return fr;
    const int fl = min(fc.ifl, c_hi + 1), ce = min(fc.ice, c_hi + 2);
    const int top = min(c_hi, ce - 1);
    fr.t_hi = min(top, fl);
    fr.a_first = max(c_lo, fl + 1);
    fr.a_last = min(c_hi + 1, ce - 1);
    return fr;
}

// One FACE JOB in a single thread (the direct path): emit(c, D) receives the signed shares.
template <int S, bool COUNT, class Emit>
__device__ __forceinline__ void face_job(PolyBuf<S> q, int c_lo, int c_hi, Emit emit, JobCounters* cnt) {
    if (COUNT) cnt->jobs++;
    const FaceClip fc = face_clip<S, true>(q);
    const FaceRun fr = face_run(fc, c_lo, c_hi);
    if (fc.n < 3 || fc.ice <= c_lo) return;
    if (COUNT) cnt->face_clips++;
    const int full_hi = min(fr.t_hi, fc.ifl - 1);  // cells entirely below Q: its projected area
    if (fc.A != 0.0)
        for (int c = c_lo; c <= full_hi; ++c) { emit(c, fc.A); if (COUNT) cnt->cells++; }
    if (fr.t_hi >= fc.ifl && fc.ifl >= c_lo) {      // the cell holding umin
        const double D = fma(-(double)fc.ifl, fc.A, fc.M1);
        if (D != 0.0) { emit(fc.ifl, D); if (COUNT) cnt->cells++; }
    }
    for (int a = fr.a_first; a <= fr.a_last; ++a) {
        const double R = plane_integral6<S>(q, fc.order, fc.n, (double)a) * (1.0 / 6.0);
        if (COUNT) cnt->plane_evals++;
        if (R != 0.0) {
            if (a <= c_hi) { emit(a, R); if (COUNT) cnt->cells++; }
            if (a - 1 >= c_lo) { emit(a - 1, -R); if (COUNT) cnt->cells++; }
        }
    }
}

}  // namespace psd

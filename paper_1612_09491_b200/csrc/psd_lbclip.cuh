// psd_lbclip.cuh -- the face triangle against the unit square of a column, without a polygon
// clipper: every boundary vertex of Q = triangle n [0,1]^2 is one of
//   (P) a point where one of the 3 triangle edges enters or leaves the square (parametric
//       Liang-Barsky clip of the edge: 4 products with the reciprocals of its (dv, dw)),
//   (V) a triangle vertex inside the square,
//   (C) a corner of the square inside the triangle;
// and going round the (counter-clockwise) triangle, the boundary of Q is
//   piece of edge 0, [corners], piece of edge 1, [corners], piece of edge 2, [corners]
// where the corners after a piece that leaves through wall k_out, up to the next piece, which
// enters through wall k_in, are the (k_in - k_out) mod 4 corners that lie counter-clockwise
// between the two walls.  All floating-point work is straight-line code over the 3 edges (no
// vertex list is edited, no wall loop); the order of the vertices is a small integer word.
//
// Every decision (edge misses the square, which wall is crossed first, vertex inside) is taken
// with a margin: when one is within PSD_LB_TOL of a tie (an edge through a corner, a vertex on a
// wall, an edge along a wall -- lattice-aligned inputs do all of these) the function reports
// "ambiguous" and the caller runs the general convex clip (clip_wall), which is consistent by
// construction.  With the margin the wall ids are those of exact arithmetic, so the cyclic
// order of the boundary points is the true one.
//
// PAPER.md:155-161 (exact tet-cube intersection); DESIGN.md section 4.
#pragma once
#include "psd_geom.cuh"

namespace psd {

#ifndef PSD_LB_TOL
#define PSD_LB_TOL 1e-10
#endif

constexpr int LB_SLOTS = 10;  // 0..5: start / end point of the piece of edge e at 2e, 2e+1; 6..9: corners

#if defined(__CUDA_ARCH__)
#define PSD_LB_RCP(x) fast_rcp(x)
#else
#define PSD_LB_RCP(x) (1.0 / (x))
#endif

// Walls in counter-clockwise order: 0: w = 0 (runs +v), 1: v = 1 (+w), 2: w = 1 (-v), 3: v = 0 (-w).
// Corner k is the start of wall k: (0,0) (1,0) (1,1) (0,1); its slot is 6 + k.
struct LBPiece {
    double t0, t1;   // kept part of the edge, 0 <= t0 < t1 <= 1
    int win, wout;   // wall entered through / left through, -1: starts / ends at a vertex inside
    bool ok;         // the edge meets the square
    bool amb;        // a decision was within the margin of a tie
};

// Parametric clip of the edge a -> b against the unit square.  One reciprocal serves both axes;
// a zero extent is replaced by 1e-150 (the edge is then inside that slab for every t or for none).
__host__ __device__ __forceinline__ LBPiece lb_edge(double va, double wa, double dv, double dw, bool a_in, bool b_in) {
    LBPiece p;
    const double dvs = dv == 0.0 ? 1e-150 : dv, dws = dw == 0.0 ? 1e-150 : dw;
    const double r = PSD_LB_RCP(dvs * dws);
    const double iv = dws * r, iw = dvs * r;               // 1 / dv, 1 / dw
    const double tlv = -va * iv, thv = tlv + iv;           // at v = 0, at v = 1
    const double tlw = -wa * iw, thw = tlw + iw;           // at w = 0, at w = 1
    const bool upv = dvs > 0.0, upw = dws > 0.0;
    const double tev = upv ? tlv : thv, txv = upv ? thv : tlv;
    const double tew = upw ? tlw : thw, txw = upw ? thw : tlw;
    const bool ev = tev > tew, xv = txv < txw;
    double t0 = ev ? tev : tew, t1 = xv ? txv : txw;
    p.win = ev ? (upv ? 3 : 1) : (upw ? 0 : 2);
    p.wout = xv ? (upv ? 1 : 3) : (upw ? 2 : 0);
    // ties: the edge's line through a corner of the square, or the edge grazing the square
    p.amb = (fabs(tev - tew) <= PSD_LB_TOL) | (fabs(txv - txw) <= PSD_LB_TOL);
    if (a_in) { t0 = 0.0; p.win = -1; }
    if (b_in) { t1 = 1.0; p.wout = -1; }
    t0 = t0 < 0.0 ? 0.0 : t0;
    t1 = t1 > 1.0 ? 1.0 : t1;
    p.ok = t0 < t1;
    p.amb = p.amb | (fabs(t1 - t0) <= PSD_LB_TOL);
    p.t0 = t0; p.t1 = t1;
    return p;
}

// Result of tri_square_clip
struct LBResult {
    unsigned order;  // nibble i = slot of vertex i (counter-clockwise)
    int n;           // vertices; 0: empty
    int sign;        // +1: as given; -1: the triangle was clockwise and has been mirrored (v -> 1 - v),
                     //     the polygon is that of the mirror image: same heights, area of opposite sign
    bool amb;        // ambiguous: nothing usable was produced, run the general clip
};

// U, V, W: the triangle's vertices, (v, w) relative to the column's lower corner.  Writes the
// piece end points into slots 0..5 and the heights of the 4 corners into slots 6..9 (the corners'
// (v, w) are constants the caller wrote once).
template <int S>
__host__ __device__ __forceinline__ LBResult tri_square_clip(PolyBuf<S> q, const double U[3], const double V[3],
                                                             const double W[3]) {
    LBResult r;
    r.order = 0; r.n = 0; r.sign = 1; r.amb = false;
    const double area2 = (V[1] - V[0]) * (W[2] - W[0]) - (V[2] - V[0]) * (W[1] - W[0]);
    if (area2 == 0.0) return r;  // the face projects to a segment: no flux through it
    // a clockwise triangle is mirrored (v -> 1 - v maps the square onto itself): counter-clockwise
    const bool ccw = area2 > 0.0;
    r.sign = ccw ? 1 : -1;
    const double ms = ccw ? 1.0 : -1.0, mo = ccw ? 0.0 : 1.0;
    double v[3];
    bool in[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        v[i] = fma(ms, V[i], mo);
        in[i] = (v[i] >= 0.0) & (v[i] <= 1.0) & (W[i] >= 0.0) & (W[i] <= 1.0);
    }
    LBPiece p[3];
    double dv[3], dw[3], du[3];
    bool amb = false;
#pragma unroll
    for (int e = 0; e < 3; ++e) {
        const int b = e == 2 ? 0 : e + 1;
        dv[e] = v[b] - v[e]; dw[e] = W[b] - W[e]; du[e] = U[b] - U[e];
        p[e] = lb_edge(v[e], W[e], dv[e], dw[e], in[e], in[b]);
        amb = amb || p[e].amb;
    }
    if (amb) { r.amb = true; return r; }
    // heights of the corners from the face's plane through vertex 0
    {
        const double inv_a = PSD_LB_RCP(fabs(area2));
        const double beta = (du[2] * dw[0] - du[0] * dw[2]) * inv_a;   // du/dv  (edges 0 and 2 leave / reach vertex 0)
        const double gamma = (dv[2] * du[0] - dv[0] * du[2]) * inv_a;  // du/dw
        const double u00 = fma(beta, -v[0], fma(gamma, -W[0], U[0]));
        q.at(6, 0) = u00;
        q.at(7, 0) = u00 + beta;
        q.at(8, 0) = u00 + beta + gamma;
        q.at(9, 0) = u00 + gamma;
    }
    if (!(p[0].ok || p[1].ok || p[2].ok)) {
        // no edge meets the square: it is inside the triangle or outside it (centre test; an edge
        // line near the centre would have given a piece)
        bool inside = true;
#pragma unroll
        for (int e = 0; e < 3; ++e) inside = inside && (dv[e] * (0.5 - W[e]) - dw[e] * (0.5 - v[e]) > 0.0);
        if (inside) { r.order = 0x9876u; r.n = 4; }
        return r;
    }
    // piece end points (stored when the piece exists) and the order word, without branches
    unsigned order = 0;
    int n = 0;
    bool bad = false;
#pragma unroll
    for (int e = 0; e < 3; ++e) {
        const int b = e == 2 ? 0 : e + 1, c = b == 2 ? 0 : b + 1;
        const bool ok = p[e].ok, starts = ok && p[e].win >= 0, endv = p[e].wout < 0;
        if (starts) {
            q.at(2 * e, 0) = fma(p[e].t0, du[e], U[e]);
            q.at(2 * e, 1) = fma(p[e].t0, dv[e], v[e]);
            q.at(2 * e, 2) = fma(p[e].t0, dw[e], W[e]);
        }
        if (ok) {
            q.at(2 * e + 1, 0) = fma(p[e].t1, du[e], U[e]);
            q.at(2 * e + 1, 1) = fma(p[e].t1, dv[e], v[e]);
            q.at(2 * e + 1, 2) = fma(p[e].t1, dw[e], W[e]);
        }
        // the next piece: it starts at this edge's end vertex, or enters through a wall
        const int kin = p[b].ok ? p[b].win : (p[c].ok ? p[c].win : p[e].win);
        bad = bad | (ok & (endv ? !(p[b].ok & (p[b].win < 0)) : (kin < 0)));
        const int cnt = (ok && !endv) ? ((kin - p[e].wout) & 3) : 0;
        // corners after wall wout, counter-clockwise: slots 6 + (wout + 1 .. wout + cnt) mod 4
        const unsigned cwd = (0x98769876u >> (4 * ((p[e].wout + 1) & 3))) & ((1u << (4 * cnt)) - 1u);
        unsigned word = starts ? (unsigned)(2 * e) | (unsigned)(2 * e + 1) << 4 : (unsigned)(2 * e + 1);
        int len = starts ? 2 : 1;
        word |= cwd << (4 * len);
        len += cnt;
        word = ok ? word : 0u;
        len = ok ? len : 0;
        order |= n < 8 ? word << (4 * n) : 0u;
        n += len;
    }
    if (bad || n > 7) { r.amb = true; return r; }
    r.order = order; r.n = n;
    return r;
}

}  // namespace psd

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
// along the third, "chord" axis u).  The triangle is clipped by the 4 axis-aligned walls of the
// column (Sutherland-Hodgman, in place) giving a convex polygon Q, on which u is linear.  With
//     R_F(a) = signed integral over Q n {u >= a} of (u - a) dv dw
// the divergence theorem (flux of (u-a,0,0)) gives, summed over the 4 faces,
//     R(a) = vol(T n column n {u >= a}),
// so the cell [a,a+1] receives R(a) - R(a+1): the cell's own faces never need a cap polygon
// (column walls have zero u-flux and the cap u = a has u-a = 0), and every face adds its own
// share to the cell independently of the other faces.  R_F(a) is evaluated in CLOSED FORM per
// fan triangle of Q (the integral of (u-a)_+ over a triangle is a cubic in a between its sorted
// vertex heights), so a lattice plane costs a few flops, not another clip.  All interpolation
// is between points on opposite sides of a plane (convex combinations), every ratio used is in
// [0,1], coordinates are local to the tile/column, arithmetic is fp64.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace psd {

constexpr int TILE = 8;            // tile edge in cells (BASELINE north_star: 8^3-cell tiles)
constexpr int TILE_CELLS = 512;
constexpr int POLY_CAP = 8;        // triangle + 4 column planes -> <= 7 vertices

// Kuhn / Freudenthal split: every tet is (corner 0, a, b, corner 7); corner index
// bit0 = +x, bit1 = +y, bit2 = +z.  Own copy (the oracle has its own).
__device__ __constant__ int c_kuhn_mid[6][2] = {{1, 3}, {5, 1}, {3, 2}, {2, 6}, {4, 5}, {6, 4}};

struct Particles {
    const void* pos;
    int dtype;   // 0 f32, 1 f64
    int stride;  // 3 or 4
    int N;
    double L;
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
__device__ __forceinline__ double unwrap1(double x, double ref, double L) {
    double d = __dsub_rn(x, ref);
    double q = __ddiv_rn(d, L);
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
        for (int x = 0; x < 3; ++x) P[v][x] = unwrap1(P[v][x], P[0][x], p.L);
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
    __device__ __forceinline__ double& at(int i, int c) { return p[(3 * i + c) * S]; }
};

// In-place Sutherland-Hodgman of a convex polygon against one wall of the column:
// AX = 1 (v) or 2 (w); UP = 0 keeps coord >= 0, UP = 1 keeps coord <= 1.  Vertices exactly on
// the plane are inside; a crossing is computed only between strictly opposite sides, always
// from the inside endpoint, so the two faces sharing a tet edge get the identical point.
template <int S, int AX, int UP>
__device__ __forceinline__ int clip_wall(PolyBuf<S> q, int n) {
    if (n == 0) return 0;
    int m = 0;
    double pu = q.at(n - 1, 0), pv = q.at(n - 1, 1), pw = q.at(n - 1, 2);
    double dp = UP ? 1.0 - (AX == 1 ? pv : pw) : (AX == 1 ? pv : pw);
    double nu = q.at(0, 0), nv = q.at(0, 1), nw = q.at(0, 2);
    for (int i = 0; i < n; ++i) {
        double cu = nu, cv = nv, cw = nw;
        if (i + 1 < n) { nu = q.at(i + 1, 0); nv = q.at(i + 1, 1); nw = q.at(i + 1, 2); }
        double dc = UP ? 1.0 - (AX == 1 ? cv : cw) : (AX == 1 ? cv : cw);
        bool pin = dp >= 0.0, cin = dc >= 0.0;
        if (pin != cin) {
            double iu = pin ? pu : cu, iv = pin ? pv : cv, iw = pin ? pw : cw;
            double ou = pin ? cu : pu, ov = pin ? cv : pv, ow = pin ? cw : pw;
            double di = pin ? dp : dc, dout = pin ? dc : dp;
            double t = di * fast_rcp(di - dout);
            double xu = fma(t, ou - iu, iu), xv = fma(t, ov - iv, iv), xw = fma(t, ow - iw, iw);
            if (AX == 1) xv = UP ? 1.0 : 0.0; else xw = UP ? 1.0 : 0.0;
            q.at(m, 0) = xu; q.at(m, 1) = xv; q.at(m, 2) = xw;
            ++m;
        }
        if (cin) {
            q.at(m, 0) = cu; q.at(m, 1) = cv; q.at(m, 2) = cw;
            ++m;
        }
        pu = cu; pv = cv; pw = cw; dp = dc;
    }
    return m;
}

// integral over a triangle of (u - a)_+ dv dw per unit (signed) area, for a lattice plane a
// strictly between the triangle's lowest and highest vertex; ua, ub, uc are the vertex heights.
// Sorted u0 <= u1 <= u2:  a >= u1: the part above is the corner triangle at u2, similar with
// ratios t/(u2-u1), t/(u2-u0), t = u2-a, mean height t/3.  a < u1: whole minus the part below,
// the corner triangle at u0.  Both ratios are in [0,1]: no cancellation, no blow-up.
__device__ __forceinline__ double tri_above_unit(double ua, double ub, double uc, double a) {
    const double lo_ab = fmin(ua, ub), hi_ab = fmax(ua, ub);
    const double u0 = fmin(lo_ab, uc), u2 = fmax(hi_ab, uc);
    const double u1 = fmax(lo_ab, fmin(hi_ab, uc));
    const double lin = (ua + ub + uc) * (1.0 / 3.0) - a;
    if (a <= u0) return lin;
    if (a >= u2) return 0.0;
    const bool hi = a >= u1;
    const double t = hi ? u2 - a : a - u0;
    const double d1 = hi ? u2 - u1 : u1 - u0;
    const double cub = t * t * t * fast_rcp(fmax(3.0 * d1 * (u2 - u0), 1e-290));
    return hi ? cub : lin + cub;
}

struct JobCounters {
    unsigned int jobs, face_clips, plane_evals, cells;
};

// faces of tet (0,1,2,3) with outward orientation when det > 0: (1,2,3) (0,3,2) (0,1,3) (0,2,1)
// packed 2 bits per vertex index, 6 bits per face.
constexpr unsigned FACE_TABLE = (1u | 2u << 2 | 3u << 4) | (0u | 3u << 2 | 2u << 4) << 6 |
                                (0u | 1u << 2 | 3u << 4) << 12 | (0u | 2u << 2 | 1u << 4) << 18;

// One FACE JOB.  q holds the face triangle: 3 vertices (u, v, w) with v, w relative to the
// column's lower corner (the column is the unit square [0,1]^2) and u in the coordinates of the
// cell run: the run is the cells c_lo..c_hi, cell c spanning u in [c, c+1].
// emit(c, D) receives the face's signed share D of the overlap volume of cell c (cell units):
//     D = R_F(c) - R_F(c+1),   R_F(a) = integral over Q n {u >= a} of (u - a) dv dw,
// Q = triangle n column.  Cells entirely below Q get the signed projected area of Q (the faces
// of the tet above and below them cancel), cells entirely above Q get nothing.
template <int S, bool COUNT, class Emit>
__device__ __forceinline__ void face_job(PolyBuf<S> q, int c_lo, int c_hi, Emit emit, JobCounters* cnt) {
    if (COUNT) cnt->jobs++;
    double minv = 1e300, maxv = -1e300, minw = 1e300, maxw = -1e300;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        double v = q.at(i, 1), w = q.at(i, 2);
        minv = fmin(minv, v); maxv = fmax(maxv, v);
        minw = fmin(minw, w); maxw = fmax(maxw, w);
    }
    if (maxv <= 0.0 || minv >= 1.0 || maxw <= 0.0 || minw >= 1.0) return;
    int n = 3;
    if (minv < 0.0) n = clip_wall<S, 1, 0>(q, n);
    if (maxv > 1.0) n = clip_wall<S, 1, 1>(q, n);
    if (minw < 0.0) n = clip_wall<S, 2, 0>(q, n);
    if (maxw > 1.0) n = clip_wall<S, 2, 1>(q, n);
    if (n < 3) return;
    // signed projected area A and first moment M1 = integral of u over Q, fan from vertex 0
    const double u0 = q.at(0, 0), v0 = q.at(0, 1), w0 = q.at(0, 2);
    double lu = q.at(1, 0), lv = q.at(1, 1), lw = q.at(1, 2);
    double umin = fmin(u0, lu), umax = fmax(u0, lu), A2 = 0.0, M6 = 0.0;
    for (int i = 2; i < n; ++i) {
        double cu = q.at(i, 0), cv = q.at(i, 1), cw = q.at(i, 2);
        double cr = (lv - v0) * (cw - w0) - (lw - w0) * (cv - v0);
        A2 += cr;
        M6 = fma(cr, u0 + lu + cu, M6);
        umin = fmin(umin, cu); umax = fmax(umax, cu);
        lu = cu; lv = cv; lw = cw;
    }
    if (umax <= (double)c_lo) return;  // entirely below the run: no share in any of its cells
    if (COUNT) cnt->face_clips++;
    const double A = 0.5 * A2, M1 = M6 * (1.0 / 6.0);
    const int top = umax >= (double)(c_hi + 1) ? c_hi : __double2int_ru(umax) - 1;
    double Rp = 0.0;
    for (int a = c_lo; a <= top + 1; ++a) {
        const double fa = (double)a;
        double R;
        if (fa <= umin) R = fma(-fa, A, M1);
        else if (fa >= umax) R = 0.0;
        else {
            // closed form per fan triangle
            double pu = q.at(1, 0), pv = q.at(1, 1), pw = q.at(1, 2), acc = 0.0;
            for (int i = 2; i < n; ++i) {
                double cu = q.at(i, 0), cv = q.at(i, 1), cw = q.at(i, 2);
                double cr = (pv - v0) * (cw - w0) - (pw - w0) * (cv - v0);
                acc = fma(cr, tri_above_unit(u0, pu, cu, fa), acc);
                pu = cu; pv = cv; pw = cw;
            }
            R = 0.5 * acc;
            if (COUNT) cnt->plane_evals++;
        }
        if (a > c_lo) {
            const double D = fa <= umin ? A : Rp - R;
            if (D != 0.0) {
                emit(a - 1, D);
                if (COUNT) cnt->cells++;
            }
        }
        Rp = R;
    }
}

}  // namespace psd

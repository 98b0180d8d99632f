// psd_faces.cuh -- the binned deposit with every face of the tessellation clipped ONCE.
//
// In the tet formulation (psd_kernels.cuh) a tet is its 4 oriented faces and each face job
// (face x column) adds  w_T * Phi(face; column, cell)  to the cells of the tet's range, Phi being
// antisymmetric in the orientation of the face.  Every face of the Lagrangian tessellation
// (the 6 tets of a cell share the cell's main diagonal) belongs to exactly two
// tets, T and N, which see it with opposite orientations, so one job can serve both:
//     cell c  +=  ( w_T [c in range of T]  -  w_N [c in range of N] ) * Phi(face; column, c)
// -- 33 % fewer clips, half the plane integrals and tile adds.  It needs one chord axis for all
// tets that add to a column (here: one axis per deposit) where the tet formulation picks the
// longest axis of each tet, which costs 30-40 % more jobs per face; the halving wins.
//
// The binning stays by (tet, tile) pair.  In the pair (T, X) a face F of T, shared with the
// neighbour N, is clipped -- once, for both tets -- if T owns F or if N does not meet tile X (then
// no pair (N, X) exists); it is skipped if N owns it and the pair (N, X) exists, which clips it
// there.  Every decision is local to the pair: what it needs of the four neighbours (determinant,
// cell range) comes from a per-tet table written once per deposit (k_tet_info).
// A tet that lies inside one cell, or is degenerate, is not deposited through its faces: its mass
// goes to its cell as the pair's "special" (its faces are still clipped where a neighbour needs them).
//
// The partial sums of a work item are no longer sums of whole tets, so they are not bounded by
// the mass of its tets: tiles and grid are accumulated in 64-bit fixed point modulo 2^64 from end
// to end (unit 2^-62 of a bound of the final cell value; integer addition commutes and wraps
// harmlessly) and the grid is converted to fp64 by a last pass (k_fixed_to_double).
//
// Measured and dropped: the same with units = the 12 faces a Lagrangian cell owns, binned by a
// census of their own (1.9x the pairs, 3.5x the binning cost: slower as a whole); a chord axis per
// tile chosen from the pairs' column counts (4 % fewer jobs: tets in a tile are not aligned).
#pragma once
#include "psd_kernels.cuh"

namespace psd {

// ---------------------------------------------------------------- the row word of one face
// The row word of ONE face (face_rows in psd_kernels.cuh does a tet's four): first row in bits
// 0..2, then 7 bits per row (first column, columns); returns the number of jobs.  pu / pv / pw:
// the 3 vertices, tile-local; lou: lowest cell (along the chord axis) that can receive anything.
// Margins as in face_rows: T = double 1e-9; T = float a margin that covers fp32's rounding.
template <typename T>
__device__ __forceinline__ int face_rows1(const double pu[3], const double pv[3], const double pw[3], const int lou,
                                          unsigned long long& rows_out) {
    using R = RowNum<T>;
    T pvv[3], pww[3], puu[3], slope[3];  // slopes of edges (0,1) (1,2) (0,2)
#pragma unroll
    for (int v = 0; v < 3; ++v) { pvv[v] = (T)pv[v]; pww[v] = (T)pw[v]; puu[v] = (T)pu[v]; }
    T smax = (T)0;
#pragma unroll
    for (int e = 0; e < 3; ++e) {
        const int i = e == 1 ? 1 : 0, j = e == 0 ? 1 : 2;
        const T dvv = pvv[j] - pvv[i];
        slope[e] = (pww[j] - pww[i]) * R::rcp(dvv == (T)0 ? (T)1 : dvv);
        if (!R::exact_rect) smax = fmax(smax, fabs(slope[e]));
    }
    T e0, em, er, erw;
    if (R::exact_rect) {
        e0 = (T)1e-9; em = (T)1e-9; er = (T)0; erw = (T)0;
    } else {
        T amax = (T)1;
#pragma unroll
        for (int v = 0; v < 3; ++v) amax = fmax(amax, fmax(fabs(puu[v]), fmax(fabs(pvv[v]), fabs(pww[v]))));
        e0 = amax * (T)0x1p-19;
        em = R::mad(e0, smax, e0);
        er = e0; erw = em;
    }
    int fv[3], cvv[3], fw[3], cww[3], cuu[3], rlo[3], rhi[3], klo[3], khi[3];
#pragma unroll
    for (int v = 0; v < 3; ++v) {
        rlo[v] = R::fl(pvv[v] - e0); rhi[v] = R::fl(pvv[v] + e0);
        klo[v] = R::fl(pww[v] - em); khi[v] = R::fl(pww[v] + em);
        if (R::exact_rect) { fv[v] = R::fl(pvv[v]); fw[v] = R::fl(pww[v]); }
        else { fv[v] = rlo[v]; fw[v] = klo[v]; }
        cvv[v] = R::ce(pvv[v] + er); cww[v] = R::ce(pww[v] + erw);
        cuu[v] = R::ce(puu[v] + er);
    }
    auto line_cols = [&](const int L, int& clo, int& chi) {
        clo = 99; chi = -99;
#pragma unroll
        for (int e = 0; e < 3; ++e) {
            const int i = e == 1 ? 1 : 0, j = e == 0 ? 1 : 2;
            const T di = pvv[i] - (T)L, dj = pvv[j] - (T)L;
            if (di * dj < (T)0) {
                const T w = R::mad(-di, slope[e], pww[i]);
                clo = min(clo, R::fl(w - em));
                chi = max(chi, R::fl(w + em));
            }
        }
    };
    const int v0 = max(min(min(fv[0], fv[1]), fv[2]), 0);
    const int v1 = min(max(max(cvv[0], cvv[1]), cvv[2]) - 1, TILE - 1);
    const int w0 = max(min(min(fw[0], fw[1]), fw[2]), 0);
    const int w1 = min(max(max(cww[0], cww[1]), cww[2]) - 1, TILE - 1);
    int c = 0;
    unsigned long long rows = 0ull;
    if (v1 >= v0 && w1 >= w0 && max(max(cuu[0], cuu[1]), cuu[2]) > lou) {
        rows = (unsigned long long)v0;
        int llo, lhi;
        line_cols(v0, llo, lhi);
#pragma unroll 1
        for (int r = v0; r <= v1; ++r) {
            int ulo, uhi;
            line_cols(r + 1, ulo, uhi);
            int rl = min(llo, ulo), rh = max(lhi, uhi);
#pragma unroll
            for (int v = 0; v < 3; ++v)
                if (rlo[v] <= r && r <= rhi[v]) { rl = min(rl, klo[v]); rh = max(rh, khi[v]); }
            const int c0 = max(rl, w0), c1 = min(rh, w1);
            const int n = max(c1 - c0 + 1, 0);
            rows |= (unsigned long long)(n ? (c0 | n << 3) : 0) << (3 + 7 * (r - v0));
            c += n;
            llo = ulo; lhi = uhi;
        }
    }
    rows_out = rows;
    return c;
}

// weight of a cell of the column: tet A's if the cell is in A's range, minus tet B's if in B's.
// cells: bit c = cell c is in A's range, bit 8 + c = in B's (range_mask)
__device__ __forceinline__ unsigned int range_mask(const int clo, const int chi) {  // clo > chi: none
    return clo <= chi ? ((2u << chi) - (1u << clo)) : 0u;
}
__device__ __forceinline__ double unit_weight(const double wA, const double wB, const unsigned int cells, const int c) {
    return ((cells >> c) & 1u ? wA : 0.0) - ((cells >> (c + 8)) & 1u ? wB : 0.0);
}

// the grid from fixed point (two's complement, unit inv_scale) to fp64, in place
__global__ void __launch_bounds__(256) k_fixed_to_double(double* grid, const long long n, const double inv_scale) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += stride) {
        const long long v = reinterpret_cast<const long long*>(grid)[i];
        grid[i] = (double)v * inv_scale;
    }
}

// ---------------------------------------------------------------- neighbours, per-tet table
// per (tet t6, face f): bits 0..5 the neighbour's Lagrangian cell as offset + 1 (2 bits per axis),
// 18 this tet owns the face (it is tet A of the face's unit), 19..21 the neighbour's t6
__device__ __constant__ unsigned int c_tet_nbr[6][4] = {
    {0x180016u, 0x140015u, 0x0c0015u, 0x240005u},
    {0x280016u, 0x000015u, 0x240015u, 0x140011u},
    {0x080019u, 0x1c0015u, 0x000015u, 0x2c0005u},
    {0x200019u, 0x2c0015u, 0x100015u, 0x040014u},
    {0x000025u, 0x080015u, 0x2c0015u, 0x1c0011u},
    {0x100025u, 0x200015u, 0x180015u, 0x0c0014u},
};

// Per tet, written once per deposit (k_tet_info) and read by the record kernel for the tet itself
// and for its four neighbours (one 16-byte load each): the tet's weight 6 m / det (0 when det = 0;
// det from the compensated determinant in the tet's own vertex order -- one number per tet wherever
// it is used; in signed-volume mode the field holds det itself), and its cell range in the image
// of its own corner 0: lo + 1024 in 12 bits per axis (bits 0..35; lo > -1024 and < 3072 for G <=
// 2048 and ranges shorter than 512), hi - lo in 9 bits per axis (36..62), bit 63: det = 0.
struct TetInfo {
    double val;
    unsigned long long box;
};
constexpr int TETINFO_MAX_EXTENT = 511;  // the host runs the tet formulation beyond
__device__ __forceinline__ int tetinfo_lo(const TetInfo& e, int x) { return (int)((e.box >> (12 * x)) & 4095ull) - 1024; }
__device__ __forceinline__ int tetinfo_ext(const TetInfo& e, int x) { return (int)((e.box >> (36 + 9 * x)) & 511ull); }
__device__ __forceinline__ bool tetinfo_one_cell(const TetInfo& e) { return ((e.box >> 36) & 0x7ffffffull) == 0ull; }
__device__ __forceinline__ bool tetinfo_degenerate(const TetInfo& e) { return (e.box >> 63) != 0ull; }
// n_levels tables, one after the other (patch mode: level l has scale0 2^l cells per box length;
// a power of two in the scale changes no rounding, so the determinant is 8^l times level 0's).
template <bool MULTI>  // false: one level (uniform grids), no loop: fewer registers
__global__ void __launch_bounds__(256) k_tet_info(Particles p, const double scale0, const int n_levels,
                                                  const double mass_per_tet, const int weight_mode, TetInfo* info) {
    const int64_t ntet = (int64_t)6 * p.N * p.N * p.N;
    const int64_t id = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (id >= ntet) return;
    double P[4][3];
    load_tet_vertices(p, id / 6, (int)(id % 6), P);
    Tet t;
    finish_tet(P, scale0, t);
    const double det0 = tet_det(t.g);
    double s2 = 1.0, s8 = 1.0;  // 2^l, 8^l
    for (int l = 0; l < (MULTI ? n_levels : 1); ++l, s2 *= 2.0, s8 *= 8.0) {
        if (l) finish_tet(P, scale0 * s2, t);
        const double det = l ? det0 * s8 : det0;
        TetInfo e;
        e.val = weight_mode == 0 ? (det != 0.0 ? 6.0 * mass_per_tet / det : 0.0) : det;
        e.box = (unsigned long long)(det == 0.0) << 63;
#pragma unroll
        for (int x = 0; x < 3; ++x)
            e.box |= (unsigned long long)((t.lo[x] + 1024) & 4095) << (12 * x) |
                     (unsigned long long)min(t.hi[x] - t.lo[x], TETINFO_MAX_EXTENT) << (36 + 9 * x);
        reinterpret_cast<double2*>(info)[(int64_t)l * ntet + id] = make_double2(e.val, __longlong_as_double((long long)e.box));
    }
}
__device__ __forceinline__ TetInfo tetinfo_load(const TetInfo* info, int64_t id) {
    const double2 v = __ldg(reinterpret_cast<const double2*>(info) + id);
    TetInfo e;
    e.val = v.x; e.box = (unsigned long long)__double_as_longlong(v.y);
    return e;
}

// a3 with the table: the scatter pass of the counting sort from the tets' cell ranges in the
// table instead of rebuilding every tet from its particles (k_census<true> does that): one thread
// per tet, the same enumeration of tiles and the same size classes as the count pass.
__global__ void __launch_bounds__(256) k_scatter_info(const TetInfo* info, const long long ntet, Space s,
                                                      const unsigned long long* tile_offsets, unsigned int* cursors,
                                                      unsigned int* pair_ids) {
    const long long id = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (id >= ntet) return;
    const int nlev = s.patch_mode ? s.n_levels : 1;
    for (int level = 0; level < nlev; ++level) {
        const TetInfo e = tetinfo_load(info + (long long)level * ntet, id);
        int lo[3], hi[3];
#pragma unroll
        for (int x = 0; x < 3; ++x) { lo[x] = tetinfo_lo(e, x); hi[x] = lo[x] + tetinfo_ext(e, x); }
        const int Gl = level_G(s, level);
        for_each_block(lo, hi, Gl, TILE, Gl / TILE, [&](int tx, int ty, int tz, long long inside) {
            const long long tid = tile_id_of(s, level, tx, ty, tz);
            if (tid < 0) return;
            const long long bin = tid * N_CLASSES + (inside > s.class_small_max ? 1 : 0);
            const unsigned int peers = __match_any_sync(__activemask(), (unsigned int)bin);
            const int leader = __ffs(peers) - 1;
            unsigned int base = 0;
            if ((int)(threadIdx.x & 31) == leader) base = atomicAdd(&cursors[bin], (unsigned int)__popc(peers));
            base = __shfl_sync(peers, base, leader);
            pair_ids[tile_offsets[bin] + base + __popc(peers & ((1u << (threadIdx.x & 31)) - 1u))] = (unsigned int)id;
        });
    }
}

// Record of a (tet, tile) pair, 23 doubles (184 bytes):
//   [0..11]  tile-local vertices (vertex v, grid axis x at 3 v + x)
//   [12]     weight of the tet, or the value of its special
//   [13..16] weights of the four neighbours (0: the neighbour adds nothing through this face here)
//   [17..20] row words of the four faces (0: the face is not clipped in this pair)
//   [21]     u64: bits 0..1 chord axis, 2 special, 3..11 its cell, 12..17 first / last cell of the tet
//            along u in the tile, 18 + 6 f .. the same of neighbour f (first > last: none)
//   [22]     jobs per face, 8 bits each
constexpr int REC2_DOUBLES = 23;
constexpr int REC2_THREADS = 128;
#ifndef REC2_MIN_CTAS
#define REC2_MIN_CTAS 5
#endif
template <int ROWS>  // 0: rows in fp64, 1: in fp32
__global__ void __launch_bounds__(REC2_THREADS, REC2_MIN_CTAS) k_pair_records2(DepositArgs A) {
    constexpr int SS = 33;
    __shared__ unsigned long long stg[REC2_THREADS / 32][REC2_DOUBLES * SS];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double* sd = reinterpret_cast<double*>(stg[warp]);
    const Item item = A.items[blockIdx.x];
    int level, org[3];
    double* out;
    long long str[3];
    tile_geometry(A.space, item.tile, level, org, out, str);
    const int G = level_G(A.space, level);
    const int ax = A.chord_axis;
    const int av = ax == 2 ? 0 : ax + 1, aw = ax == 0 ? 2 : ax - 1;
    const int N = A.part.N;
    const double scale = level_scale(A.space, level);
    // the per-tet table of this tile's level (patch mode: one table per level, cell ranges differ)
    const TetInfo* info = reinterpret_cast<const TetInfo*>(A.tet_info) + (long long)level * 6 * N * N * N;
    for (unsigned int k0 = 0; k0 < item.count; k0 += REC2_THREADS) {
        const unsigned int kk = k0 + threadIdx.x;
        __syncwarp();
        if (kk < item.count) {
            const unsigned int id = A.pair_ids[item.begin + (item.count - 1u - kk)];
            const unsigned int cell = id / 6u;
            const int t6 = (int)(id - cell * 6u);
            const int k = (int)(cell % N), j = (int)((cell / N) % N), i = (int)(cell / ((unsigned int)N * N));
            const TetInfo me = tetinfo_load(info, (int64_t)id);
            double P[4][3];
            load_tet_vertices(A.part, (int64_t)cell, t6, P);
            int lo[3], hi[3], o[3];
#pragma unroll
            for (int x = 0; x < 3; ++x) {
                lo[x] = tetinfo_lo(me, x);
                hi[x] = lo[x] + tetinfo_ext(me, x);
                o[x] = org[x] - floor_div(org[x] + TILE - 1 - lo[x], G) * G;  // the image of the tile the tet meets
#pragma unroll
                for (int v = 0; v < 4; ++v) sd[(3 * v + x) * SS + lane] = __dmul_rn(P[v][x], scale) - (double)o[x];
            }
            const bool cellT = tetinfo_one_cell(me);
            double wT = A.weight_mode == 0 ? me.val : 1.0;
            bool actT = true;
            unsigned int special = 0u, scell = 0u;
            if (tetinfo_degenerate(me)) {  // degenerate: whole mass to the centroid cell (Q6)
                actT = false;
                if (A.weight_mode == 0) {
                    int c[3];
                    bool in = true;
#pragma unroll
                    for (int x = 0; x < 3; ++x) {
                        const double cen = (__dmul_rn(P[0][x], scale) + __dmul_rn(P[1][x], scale) + __dmul_rn(P[2][x], scale) + __dmul_rn(P[3][x], scale)) / 4.0;
                        c[x] = __double2int_rd(cen) - o[x];
                        in = in && c[x] >= 0 && c[x] < TILE;
                    }
                    if (in) { special = 1u; scell = (unsigned int)((c[0] * TILE + c[1]) * TILE + c[2]); wT = A.mass_per_tet; }
                }
            } else if (cellT) {  // inside one cell: the whole tet goes to that cell
                actT = false;
                special = 1u;
                scell = (unsigned int)(((lo[0] - o[0]) * TILE + (lo[1] - o[1])) * TILE + (lo[2] - o[2]));
                wT = A.weight_mode == 0 ? A.mass_per_tet : me.val * (1.0 / 6.0);
            }
            const int loU = ax == 0 ? lo[0] : (ax == 1 ? lo[1] : lo[2]), hiU = ax == 0 ? hi[0] : (ax == 1 ? hi[1] : hi[2]);
            const int oU = ax == 0 ? o[0] : (ax == 1 ? o[1] : o[2]);
            int cloT = max(loU - oU, 0), chiT = min(hiU - oU, TILE - 1);
            if (!actT || cloT > chiT) { cloT = TILE - 1; chiT = 0; actT = false; }
            unsigned long long word = (unsigned long long)ax | (unsigned long long)special << 2 | (unsigned long long)scell << 3 |
                                      (unsigned long long)(cloT | chiT << 3) << 12;
            unsigned int cnts = 0u;
            // the four neighbours' table entries, all loads in flight before the first is used
            TetInfo nbr[4];
#pragma unroll
            for (int f = 0; f < 4; ++f) {
                const unsigned int nb = c_tet_nbr[t6][f];
                int ni = i + (int)(nb & 3u) - 1, nj = j + (int)((nb >> 2) & 3u) - 1, nk = k + (int)((nb >> 4) & 3u) - 1;
                ni = ni < 0 ? ni + N : (ni >= N ? ni - N : ni);
                nj = nj < 0 ? nj + N : (nj >= N ? nj - N : nj);
                nk = nk < 0 ? nk + N : (nk >= N ? nk - N : nk);
                nbr[f] = tetinfo_load(info, (((int64_t)ni * N + nj) * N + nk) * 6 + (int)((nb >> 19) & 7u));
            }
#pragma unroll
            for (int f = 0; f < 4; ++f) {
                const unsigned int nb = c_tet_nbr[t6][f];
                // the neighbour behind face f: its cell range in this tet's image
                const TetInfo en = nbr[f];
                int nlo[3], nhi[3];
                bool meets = true;
#pragma unroll
                for (int x = 0; x < 3; ++x) {
                    int l = tetinfo_lo(en, x);
                    const int d = lo[x] - l;      // the two tets share a face: their ranges are close
                    l += 2 * d > G ? G : (2 * d < -G ? -G : 0);
                    nlo[x] = l - o[x];
                    nhi[x] = nlo[x] + tetinfo_ext(en, x);
                    meets = meets && nlo[x] <= TILE - 1 && nhi[x] >= 0;
                }
                const bool cellN = tetinfo_one_cell(en);
                const bool own = (nb >> 18) & 1u;
                double wN = 0.0;
                int cloN = TILE - 1, chiN = 0;
                if (meets && !cellN) {
                    wN = A.weight_mode == 0 ? en.val : 1.0;
                    const int nl = ax == 0 ? nlo[0] : (ax == 1 ? nlo[1] : nlo[2]), nh = ax == 0 ? nhi[0] : (ax == 1 ? nhi[1] : nhi[2]);
                    cloN = max(nl, 0); chiN = min(nh, TILE - 1);
                    if (wN == 0.0) { cloN = TILE - 1; chiN = 0; }
                }
                const bool anyN = cloN <= chiN;
                unsigned long long rows = 0ull;
                int njobs = 0;
                if ((own || !meets) && (actT || anyN)) {
                    double pu[3], pv[3], pw[3];
#pragma unroll
                    for (int q = 0; q < 3; ++q) {
                        const int vi = (int)((FACE_TABLE >> (6 * f + 2 * q)) & 3u);
                        pu[q] = sd[(3 * vi + ax) * SS + lane];
                        pv[q] = sd[(3 * vi + av) * SS + lane];
                        pw[q] = sd[(3 * vi + aw) * SS + lane];
                    }
                    const int lou = actT ? (anyN ? min(cloT, cloN) : cloT) : cloN;
                    njobs = ROWS ? face_rows1<float>(pu, pv, pw, lou, rows) : face_rows1<double>(pu, pv, pw, lou, rows);
                }
                sd[(13 + f) * SS + lane] = wN;
                stg[warp][(17 + f) * SS + lane] = rows;
                word |= (unsigned long long)(cloN | chiN << 3) << (18 + 6 * f);
                cnts |= (unsigned int)njobs << (8 * f);
            }
            sd[12 * SS + lane] = wT;
            stg[warp][21 * SS + lane] = word;
            stg[warp][22 * SS + lane] = (unsigned long long)cnts;
        }
        __syncwarp();
        const unsigned int kw = k0 + 32u * warp;
        if (kw < item.count) {
            const int valid = (int)min(32u, item.count - kw);
            unsigned long long* dst = reinterpret_cast<unsigned long long*>(const_cast<double*>(A.rec_g)) +
                                      ((long long)(item.begin - A.rec_pair_begin) + kw) * REC2_DOUBLES;
#pragma unroll
            for (int q = 0; q < REC2_DOUBLES; ++q) {
                const int d = q * 32 + lane;
                const int jr = (d * 2850) >> 16;  // d / 23 for d < 736
                const int c = d - jr * REC2_DOUBLES;
                if (jr < valid) dst[d] = stg[warp][c * SS + jr];
            }
        }
    }
}

__device__ __forceinline__ double rec2_d(const DepositArgs& A, long long r, int c) { return __ldg(A.rec_g + r * REC2_DOUBLES + c); }
__device__ __forceinline__ unsigned long long rec2_u(const DepositArgs& A, long long r, int c) {
    return __ldg(reinterpret_cast<const unsigned long long*>(A.rec_g) + r * REC2_DOUBLES + c);
}
// As k_deposit_tiles<COUNT, true> on the records of k_pair_records2: four faces per slot, each with
// the weight and range of the neighbour behind it; the tile is flushed as 64-bit integers.
#ifndef DEP2_MIN_CTAS
#define DEP2_MIN_CTAS 6
#endif
template <bool COUNT>
__global__ void __launch_bounds__(DEP_THREADS, DEP2_MIN_CTAS) k_deposit_tiles2(DepositArgs A) {
    extern __shared__ double smem[];
    double* acc = smem;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double* wpoly = smem + TILE_CELLS + warp * WARP_SCRATCH_REC;  // [3 * LB_SLOTS][32]
    PolyBuf<32> poly{wpoly + lane};
    poly.at(6, 1) = 0.0; poly.at(6, 2) = 0.0; poly.at(7, 1) = 1.0; poly.at(7, 2) = 0.0;
    poly.at(8, 1) = 1.0; poly.at(8, 2) = 1.0; poly.at(9, 1) = 0.0; poly.at(9, 2) = 1.0;
    bool slot6_dirty = false;

    const Item item = A.items[blockIdx.x];
    int level, org[3];
    double* out;
    long long str[3];
    tile_geometry(A.space, item.tile, level, org, out, str);
    const int ax = A.chord_axis;
    const int av = ax == 2 ? 0 : ax + 1, aw = ax == 0 ? 2 : ax - 1;
    const int su = ax == 0 ? 64 : (ax == 1 ? 8 : 1), sv = av == 0 ? 64 : (av == 1 ? 8 : 1), sw = aw == 0 ? 64 : (aw == 1 ? 8 : 1);

    __shared__ unsigned int sh_next;
    for (int i = threadIdx.x; i < TILE_CELLS; i += DEP_THREADS) acc[i] = 0.0;
    if (threadIdx.x == 0) sh_next = 0u;
    __syncthreads();
    JobCounters cnt = {0, 0, 0, 0, 0};

    for (;;) {
        unsigned int base = 0;
        if (lane == 0) base = atomicAdd(&sh_next, 32u);
        base = __shfl_sync(0xffffffffu, base, 0);
        if (base >= item.count) break;
        const bool have = base + lane < item.count;
        const long long rb = (long long)(item.begin - A.rec_pair_begin) + base;
        int njobs = 0;
        unsigned int cnts = 0u;
        if (have) {
            asm volatile("prefetch.global.L1 [%0];" ::"l"(A.rec_g + (rb + lane) * REC2_DOUBLES));
            asm volatile("prefetch.global.L1 [%0];" ::"l"(A.rec_g + (rb + lane) * REC2_DOUBLES + 16));
            const unsigned int word = (unsigned int)rec2_u(A, rb + lane, 21);
            cnts = (unsigned int)rec2_u(A, rb + lane, 22);
            njobs = (int)((cnts & 255u) + ((cnts >> 8) & 255u) + ((cnts >> 16) & 255u) + (cnts >> 24));
            if ((word >> 2) & 1u) tile_add(acc, (int)((word >> 3) & 511u), tile_share(rec2_d(A, rb + lane, 12), A.acc_scale));
        }
        int pre = njobs;
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(0xffffffffu, pre, o);
            if (lane >= o) pre += y;
        }
        const int total = __shfl_sync(0xffffffffu, pre, 31);
        pre -= njobs;
#pragma unroll 1
        for (int jb = 0; jb < total; jb += 32) {
            const int job = jb + lane;
            int slot = 0;
#pragma unroll
            for (int step = 16; step; step >>= 1) {
                int probe = __shfl_sync(0xffffffffu, pre, slot + step);
                if (probe <= job) slot += step;
            }
            const int spre = __shfl_sync(0xffffffffu, pre, slot);
            const unsigned int scnt = __shfl_sync(0xffffffffu, cnts, slot);
            const bool act = job < total;
            unsigned int f_order = 0, f_info = 0, f_floors = 0, f_aux = 0;
            int kpl = 0;
            double f_wA = 0.0, f_wB = 0.0;
            if (act) {
                if (COUNT) cnt.jobs++;
                const long long rs = rb + slot;
                // (face, row, column) of the job: the slot's four face counts, then the face's row word
                int local = job - spre, f = 0;
                unsigned int sc = scnt;
#pragma unroll
                for (int q = 0; q < 3; ++q) {
                    const int n = (int)(sc & 255u);
                    if (local < n) break;
                    local -= n; ++f; sc >>= 8;
                }
                unsigned long long rw = rec2_u(A, rs, 17 + f);
                int cv = (int)(rw & 7ull);
                rw >>= 3;
#pragma unroll
                for (int r = 0; r < TILE; ++r) {
                    const int n = (int)(rw >> 3) & 15;
                    if (local < n) break;
                    local -= n; ++cv; rw >>= 7;
                }
                const int cw = ((int)rw & 7) + local;
                const unsigned long long word = rec2_u(A, rs, 21);
                const unsigned int rng = (unsigned int)((word >> 12) & 63ull) | (unsigned int)((word >> (18 + 6 * f)) & 63ull) << 6;
                const bool spc = (word >> 2) & 1ull;
                const int cloA = rng & 7, chiA = (rng >> 3) & 7, cloB = (rng >> 6) & 7, chiB = (rng >> 9) & 7;
                const unsigned int cells = range_mask(cloA, chiA) | range_mask(cloB, chiB) << 8;
                const bool anyA = cloA <= chiA, anyB = cloB <= chiB;
                const int c_lo = anyA ? (anyB ? min(cloA, cloB) : cloA) : cloB;
                const int c_hi = anyA ? (anyB ? max(chiA, chiB) : chiA) : chiB;
                const double ov = (double)cv, ow = (double)cw;
                double U[3], V[3], W[3];
#pragma unroll
                const unsigned int fvt = FACE_TABLE >> (6 * f);
#pragma unroll
                for (int i = 0; i < 3; ++i) {
                    const int vi = (fvt >> (2 * i)) & 3;
                    U[i] = rec2_d(A, rs, 3 * vi + ax);
                    V[i] = rec2_d(A, rs, 3 * vi + av) - ov;
                    W[i] = rec2_d(A, rs, 3 * vi + aw) - ow;
                }
                double wA = spc ? 0.0 : rec2_d(A, rs, 12), wB = rec2_d(A, rs, 13 + f);
                if (slot6_dirty) { poly.at(6, 1) = 0.0; poly.at(6, 2) = 0.0; slot6_dirty = false; }
                const LBResult lb = tri_square_clip<32>(poly, U, V, W);
                FaceClip fc;
                if (lb.amb) {
#pragma unroll
                    for (int i = 0; i < 3; ++i) { poly.at(i, 0) = U[i]; poly.at(i, 1) = V[i]; poly.at(i, 2) = W[i]; }
                    fc = face_clip_general(wpoly + lane);
                    slot6_dirty = true;
                    if (COUNT) cnt.general++;
                } else {
                    fc = poly_area_moment<32>(poly, lb.order, lb.n);
                    if (lb.sign < 0) { wA = -wA; wB = -wB; }
                }
                if (fc.n >= 3 && fc.ice > c_lo) {
                    if (COUNT) cnt.face_clips++;
                    const FaceRun fr = face_run(fc, c_lo, c_hi);
                    const int colofs = cv * sv + cw * sw;
                    {
                        const int full_hi = min(fr.t_hi, fc.ifl - 1);  // cells entirely below Q
                        if (fc.A != 0.0) {
#pragma unroll
                            for (int cc = 0; cc < TILE; ++cc) {
                                const int c = c_lo + cc;
                                if (c > full_hi) break;
                                const double wc = unit_weight(wA, wB, cells, c);
                                if (wc != 0.0) {
                                    tile_add(acc, colofs + c * su, tile_share(wc * fc.A, A.acc_scale));
                                    if (COUNT) cnt.cells++;
                                }
                            }
                        }
                        if (fr.t_hi >= fc.ifl && fc.ifl >= c_lo) {  // the cell holding umin
                            const double D = fma(-(double)fc.ifl, fc.A, fc.M1) * unit_weight(wA, wB, cells, fc.ifl);
                            if (D != 0.0) {
                                tile_add(acc, colofs + fc.ifl * su, tile_share(D, A.acc_scale));
                                if (COUNT) cnt.cells++;
                            }
                        }
                    }
                    kpl = max(fr.a_last - fr.a_first + 1, 0);
                    f_order = fc.order;
                    f_floors = fc.floors;
                    f_aux = (unsigned)fr.a_first | cells << 4;
                    f_info = (unsigned)colofs | (unsigned)c_lo << 11 | (unsigned)c_hi << 14 | (unsigned)fc.n << 17 | fc.below0 << 20;
                    f_wA = wA; f_wB = wB;
                }
            }
            __syncwarp();
            // ---- the cutting planes of the 32 polygons, lane = plane
            int pre2 = kpl;
            for (int o = 1; o < 32; o <<= 1) {
                int y = __shfl_up_sync(0xffffffffu, pre2, o);
                if (lane >= o) pre2 += y;
            }
            const int total2 = __shfl_sync(0xffffffffu, pre2, 31);
            pre2 -= kpl;
            for (int eb = 0; eb < total2; eb += 32) {
                const int e = eb + lane;
                int src = 0;
#pragma unroll
                for (int step = 16; step; step >>= 1) {
                    int probe = __shfl_sync(0xffffffffu, pre2, src + step);
                    if (probe <= e) src += step;
                }
                const int s_pre = __shfl_sync(0xffffffffu, pre2, src);
                const unsigned int s_order = __shfl_sync(0xffffffffu, f_order, src);
                const unsigned int s_info = __shfl_sync(0xffffffffu, f_info, src);
                const unsigned int s_floors = __shfl_sync(0xffffffffu, f_floors, src);
                const unsigned int s_aux = __shfl_sync(0xffffffffu, f_aux, src);
                const double s_wA = __shfl_sync(0xffffffffu, f_wA, src);
                const double s_wB = __shfl_sync(0xffffffffu, f_wB, src);
                if (e < total2) {
                    const int a = (int)(s_aux & 15u) + (e - s_pre);
                    const unsigned int cells = s_aux >> 4;
                    const int colofs = s_info & 511;
                    const int c_lo = (s_info >> 11) & 7, c_hi = (s_info >> 14) & 7, n = (s_info >> 17) & 7;
                    PolyBuf<32> qs{wpoly + src};
                    const double R = plane_integral6_mask<32>(qs, s_order, n, (double)a, plane_mask_from_floors(s_floors, (s_info >> 20) & 127u, n, a)) * (1.0 / 6.0);
                    if (COUNT) cnt.plane_evals++;
                    if (R != 0.0) {
                        if (a <= c_hi) {
                            const double x = R * unit_weight(s_wA, s_wB, cells, a);
                            if (x != 0.0) { tile_add(acc, colofs + a * su, tile_share(x, A.acc_scale)); if (COUNT) cnt.cells++; }
                        }
                        if (a - 1 >= c_lo) {
                            const double x = -R * unit_weight(s_wA, s_wB, cells, a - 1);
                            if (x != 0.0) { tile_add(acc, colofs + (a - 1) * su, tile_share(x, A.acc_scale)); if (COUNT) cnt.cells++; }
                        }
                    }
                }
            }
            __syncwarp();
        }
    }
    __syncthreads();
    // ---- flush: 64-bit integer reductions (modulo 2^64), the grid is in fixed point for now
    {
        const unsigned int* a = reinterpret_cast<const unsigned int*>(acc);
        unsigned long long* o64 = reinterpret_cast<unsigned long long*>(out);
        for (int i = threadIdx.x; i < TILE_CELLS; i += DEP_THREADS) {
            const unsigned long long v = ((unsigned long long)a[TILE_CELLS + i] << 32) | a[i];
            if (v) {
                int cz = i & 7, cy = (i >> 3) & 7, cx = i >> 6;
                atomicAdd(o64 + cx * str[0] + cy * str[1] + cz, v);
            }
        }
    }
    if (COUNT) {
        unsigned int a = __reduce_add_sync(0xffffffffu, cnt.jobs), b = __reduce_add_sync(0xffffffffu, cnt.face_clips);
        unsigned int c = __reduce_add_sync(0xffffffffu, cnt.plane_evals), d = __reduce_add_sync(0xffffffffu, cnt.cells);
        const unsigned int e = __reduce_add_sync(0xffffffffu, cnt.general);
        if (lane == 0) {
            atomicAdd(&A.stats[ST_TASKS], (unsigned long long)a);
            atomicAdd(&A.stats[ST_FACE_CLIPS], (unsigned long long)b);
            atomicAdd(&A.stats[ST_PLANE_CLIPS], (unsigned long long)c);
            atomicAdd(&A.stats[ST_CELLS], (unsigned long long)d);
            if (e) atomicAdd(&A.stats[ST_GENERAL], (unsigned long long)e);
        }
    }
}


}  // namespace psd

// psd_kernels.cuh -- kernels of the deposit path (sm_100a).  Steps:
//   a1 tet generation        load_tet_vertices, inlined where a tet is needed (nothing stored per tet)
//   a2 AABB + census         k_census<false> (pair counts per (tile, size class), histograms)
//   a3 bin / sort            k_scan_* + k_census<true> (counting sort of tet ids by tile and class) + k_items
//   a3' per-pair stage A     stage_a / k_pair_records (tile-local vertices, weight, per-row column
//                            ranges of the faces -> 144-byte pair records), k_slab_bounds
//   a4-a6 classify, clip, accumulate, flush    k_deposit_tiles (binned) / k_deposit_direct
//   a7 patch path            the same kernels with Space::patch_mode = 1, k_patch_counts,
//                            k_subblock_counts, k_restrict
#pragma once
#include "psd_geom.cuh"
#include "psd_lbclip.cuh"

namespace psd {

struct PatchDev { int level, ox, oy, oz; };

// Where deposits go: a uniform periodic G^3 grid, or a list of P^3 patches on level grids.
struct Space {
    int patch_mode;
    // uniform
    int G;            // cells per side
    int nt;           // tiles per side (G/8), binned path only
    // patches
    int base_G, P, tp;        // tp = P/8 tiles per patch side
    int tp_shift, np0;        // log2(tp) or -1; np0 = base_G / P patch positions per side on level 0
    int n_levels;
    const PatchDev* patches;  // device
    const int* lookup;        // dense patch-position -> patch index (or -1), levels concatenated
    long long lookup_off[8];  // start of each level in lookup
    double* out;
    double L;
    long long class_small_max;  // a3: pairs covering at most this many cells of the tile are class "small"
};

__device__ __forceinline__ double level_scale(const Space& s, int level) {
    return s.patch_mode ? __ddiv_rn((double)(s.base_G << level), s.L) : __ddiv_rn((double)s.G, s.L);
}
__device__ __forceinline__ int level_G(const Space& s, int level) {
    return s.patch_mode ? (s.base_G << level) : s.G;
}

struct Item { unsigned int tile; unsigned int count; unsigned long long begin; };

// a3: every tile's pair list is ordered by SIZE CLASS of the pair -- class 0 "small": the tet's
// cell range covers <= 8 cells of the tile (buckets b <= 3 of the census histogram), class 1
// "large" -- so the 32-pair batches a warp fetches hold tets of similar size.  Bin = tile * 2 + class.
constexpr int N_CLASSES = 2;
constexpr long long CLASS_SMALL_MAX_CELLS = 8;  // default of PSD_OPT_CLASS_SMALL_CELLS

enum { ST_SUM_CELLS = 0, ST_MAX_CELLS, ST_INVERTED, ST_DEGENERATE, ST_UNWRAP, ST_NONFINITE,
       ST_PAIRS, ST_TASKS, ST_FACE_CLIPS, ST_PLANE_CLIPS, ST_CELLS, ST_GENERAL, ST_MAX_EXTENT, ST_ROWS_MISSED, ST_COUNT };

// ---------------------------------------------------------------- validation of positions
__global__ void k_validate(Particles p, unsigned long long* stats) {
    int64_t n = (int64_t)p.N * p.N * p.N;
    unsigned int bad = 0;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
        double v[3];
        load_pos(p, i, v);
        bad += !(isfinite(v[0]) && isfinite(v[1]) && isfinite(v[2]));
    }
    bad = __reduce_add_sync(0xffffffffu, bad);
    if ((threadIdx.x & 31) == 0 && bad) atomicAdd(&stats[ST_NONFINITE], (unsigned long long)bad);
}

// Enumerate the distinct periodic blocks (edge `bs` cells, `nb` per side) met by the cell range
// [lo,hi] of one tet on a grid of Gl cells; f(bx,by,bz, cells_inside) once per block.
template <class F>
__device__ __forceinline__ void for_each_block(const int lo[3], const int hi[3], int Gl, int bs,
                                               int nb, F f) {
    int b0[3], cnt[3];
#pragma unroll
    for (int x = 0; x < 3; ++x) {
        b0[x] = floor_div(lo[x], bs);
        cnt[x] = min(floor_div(hi[x], bs) - b0[x] + 1, nb);
    }
    // common case: the range is short enough on every axis to meet each block in one periodic
    // image only -> no division, the per-axis terms hoisted out of the inner loops
    if (hi[0] - lo[0] < Gl - bs && hi[1] - lo[1] < Gl - bs && hi[2] - lo[2] < Gl - bs) {
        auto wrap1 = [nb](int v) {
            int r = v < 0 ? v + nb : (v >= nb ? v - nb : v);
            return (unsigned)r < (unsigned)nb ? r : wrap_mod(v, nb);
        };
        auto cells = [bs](int l, int h, int b) { return min(h, b * bs + bs - 1) - max(l, b * bs) + 1; };
        for (int qx = 0; qx < cnt[0]; ++qx) {
            const int bx = wrap1(b0[0] + qx), cx = cells(lo[0], hi[0], b0[0] + qx);
            for (int qy = 0; qy < cnt[1]; ++qy) {
                const int by = wrap1(b0[1] + qy), cxy = cx * cells(lo[1], hi[1], b0[1] + qy);
                for (int qz = 0; qz < cnt[2]; ++qz)
                    f(bx, by, wrap1(b0[2] + qz), (long long)cxy * cells(lo[2], hi[2], b0[2] + qz));
            }
        }
        return;
    }
    for (int qx = 0; qx < cnt[0]; ++qx)
        for (int qy = 0; qy < cnt[1]; ++qy)
            for (int qz = 0; qz < cnt[2]; ++qz) {
                int q[3] = {qx, qy, qz}, bw[3];
                long long inside = 1;
#pragma unroll
                for (int x = 0; x < 3; ++x) {
                    bw[x] = wrap_mod(b0[x] + q[x], nb);
                    // cells of [lo,hi] whose wrapped position falls in block bw (all images)
                    int first = bw[x] * bs;
                    int m_lo = -floor_div(first + bs - 1 - lo[x], Gl);  // ceil((lo-first-bs+1)/Gl)
                    int m_hi = floor_div(hi[x] - first, Gl);
                    int c = 0;
                    for (int m = m_lo; m <= m_hi; ++m) {
                        int a = max(lo[x], first + m * Gl), b = min(hi[x], first + bs - 1 + m * Gl);
                        c += max(b - a + 1, 0);
                    }
                    inside *= c;
                }
                f(bw[0], bw[1], bw[2], inside);
            }
}

// tile id of wrapped tile coords on `level`; -1 if no patch there (patch mode)
__device__ __forceinline__ long long tile_id_of(const Space& s, int level, int tx, int ty, int tz) {
    if (!s.patch_mode) return ((long long)tx * s.nt + ty) * s.nt + tz;
    const int np = s.np0 << level;  // patch positions per side: (base_G / P) * 2^level
    int px, py, pz, sx, sy, sz;
    if (s.tp_shift >= 0) {  // tiles per patch side a power of two: no integer division
        const int m = s.tp - 1;
        px = tx >> s.tp_shift; py = ty >> s.tp_shift; pz = tz >> s.tp_shift;
        sx = tx & m; sy = ty & m; sz = tz & m;
    } else {
        px = tx / s.tp; py = ty / s.tp; pz = tz / s.tp;
        sx = tx - px * s.tp; sy = ty - py * s.tp; sz = tz - pz * s.tp;
    }
    const int pi = s.lookup[s.lookup_off[level] + ((long long)px * np + py) * np + pz];
    if (pi < 0) return -1;
    return (long long)pi * (s.tp * s.tp * s.tp) + (sx * s.tp + sy) * s.tp + sz;
}

// ---------------------------------------------------------------- a2 census / a3 scatter
// One thread per Lagrangian cell (6 tets).  SCATTER = false: count pairs per tile + statistics.
// SCATTER = true: write tet ids into the per-tile lists (counting sort, order within a tile is
// the arrival order of the atomics).
template <bool SCATTER>
__global__ void __launch_bounds__(256) k_census(Particles p, Space s, unsigned int* tile_counts,
                                                const unsigned long long* tile_offsets,
                                                unsigned int* cursors, unsigned int* pair_ids,
                                                unsigned long long* stats,
                                                unsigned long long* hist /* [2][64] */) {
    __shared__ unsigned int sh_hist[2][64];
    __shared__ unsigned long long sh_stat[ST_COUNT];
    if (!SCATTER) {
        for (int i = threadIdx.x; i < 128; i += blockDim.x) (&sh_hist[0][0])[i] = 0;
        if (threadIdx.x < ST_COUNT) sh_stat[threadIdx.x] = 0;
        __syncthreads();
    }
    const int N = p.N;
    const int64_t ncell = (int64_t)N * N * N;
    int64_t cell = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    // statistics are summed per thread over its 6 tets, then per warp, then one shared atomic each
    unsigned long long t_sum = 0, t_max = 0;
    unsigned int t_inv = 0, t_deg = 0, t_pairs = 0, t_suspect = 0, t_ext = 0;
    if (cell < ncell) {
        int k = (int)(cell % N), j = (int)((cell / N) % N), i = (int)(cell / ((int64_t)N * N));
        double C[8][3];
#pragma unroll
        for (int b = 0; b < 8; ++b) load_pos(p, corner_index(i, j, k, b, N), C[b]);
        unsigned int suspect = 0;
#pragma unroll
        for (int b = 1; b < 8; ++b)
#pragma unroll
            for (int x = 0; x < 3; ++x) {
                C[b][x] = unwrap1(C[b][x], C[0][x], p.L, p.inv_L);
                if (!SCATTER && (b == 1 || b == 2 || b == 4))
                    suspect |= fabs(C[b][x] - C[0][x]) > 0.25 * p.L;
            }
        t_suspect = suspect;
        const int nlev = s.patch_mode ? s.n_levels : 1;
        for (int level = 0; level < nlev; ++level) {
            const double scale = level_scale(s, level);
            const int Gl = level_G(s, level);
            const int nb = Gl / TILE;
#pragma unroll 1
            for (int t6 = 0; t6 < 6; ++t6) {
                double P[4][3];
                int ca = c_kuhn_mid[t6][0], cb = c_kuhn_mid[t6][1];
#pragma unroll
                for (int x = 0; x < 3; ++x) {
                    P[0][x] = C[0][x]; P[1][x] = C[ca][x]; P[2][x] = C[cb][x]; P[3][x] = C[7][x];
                }
                Tet t;
                finish_tet(P, scale, t);
                unsigned int tet_id = (unsigned int)(cell * 6 + t6);
                if (!SCATTER && level == 0) {
                    long long nc = (long long)(t.hi[0] - t.lo[0] + 1) * (t.hi[1] - t.lo[1] + 1) *
                                   (t.hi[2] - t.lo[2] + 1);
                    t_sum += (unsigned long long)nc;
                    t_max = (unsigned long long)nc > t_max ? (unsigned long long)nc : t_max;
                    t_ext = max(t_ext, (unsigned int)max(max(t.hi[0] - t.lo[0], t.hi[1] - t.lo[1]), t.hi[2] - t.lo[2]) + 1u);
                    atomicAdd(&sh_hist[0][bit_width_u64((unsigned long long)(nc - 1))], 1u);
                    double det = tet_det_sign(t.g);
                    t_inv += det < 0.0;
                    t_deg += det == 0.0;
                }
                for_each_block(t.lo, t.hi, Gl, TILE, nb, [&](int tx, int ty, int tz, long long inside) {
                    long long id = tile_id_of(s, level, tx, ty, tz);
                    if (id < 0) return;
                    // size class of the pair: cells of the tet's range inside this tile (a3)
                    const long long bin = id * N_CLASSES + (inside > s.class_small_max ? 1 : 0);
                    if (!SCATTER) {
                        const unsigned int peers = __match_any_sync(__activemask(), (unsigned int)bin);
                        if ((int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(&tile_counts[bin], (unsigned int)__popc(peers));
                        ++t_pairs;
                        atomicAdd(&sh_hist[1][bit_width_u64((unsigned long long)(inside - 1))], 1u);
                    } else {
                        // one cursor atomic per distinct bin among the lanes that are here together
                        const unsigned int peers = __match_any_sync(__activemask(), (unsigned int)bin);
                        const int leader = __ffs(peers) - 1;
                        unsigned int base = 0;
                        if ((int)(threadIdx.x & 31) == leader) base = atomicAdd(&cursors[bin], (unsigned int)__popc(peers));
                        base = __shfl_sync(peers, base, leader);
                        const unsigned int slot = base + __popc(peers & ((1u << (threadIdx.x & 31)) - 1u));
                        pair_ids[tile_offsets[bin] + slot] = tet_id;
                    }
                });
            }
        }
    }
    if (!SCATTER) {
        for (int o = 16; o; o >>= 1) {
            t_sum += __shfl_down_sync(0xffffffffu, t_sum, o);
            const unsigned long long y = __shfl_down_sync(0xffffffffu, t_max, o);
            t_max = y > t_max ? y : t_max;
        }
        t_inv = __reduce_add_sync(0xffffffffu, t_inv);
        t_deg = __reduce_add_sync(0xffffffffu, t_deg);
        t_pairs = __reduce_add_sync(0xffffffffu, t_pairs);
        t_suspect = __reduce_add_sync(0xffffffffu, t_suspect);
        t_ext = __reduce_max_sync(0xffffffffu, t_ext);
        if ((threadIdx.x & 31) == 0) {
            atomicMax(&sh_stat[ST_MAX_EXTENT], (unsigned long long)t_ext);
            atomicAdd(&sh_stat[ST_SUM_CELLS], t_sum);
            atomicMax(&sh_stat[ST_MAX_CELLS], t_max);
            if (t_inv) atomicAdd(&sh_stat[ST_INVERTED], (unsigned long long)t_inv);
            if (t_deg) atomicAdd(&sh_stat[ST_DEGENERATE], (unsigned long long)t_deg);
            if (t_pairs) atomicAdd(&sh_stat[ST_PAIRS], (unsigned long long)t_pairs);
            if (t_suspect) atomicAdd(&sh_stat[ST_UNWRAP], (unsigned long long)t_suspect);
        }
        __syncthreads();
        for (int i = threadIdx.x; i < 128; i += blockDim.x) {
            unsigned int v = (&sh_hist[0][0])[i];
            if (v) atomicAdd(&hist[i], (unsigned long long)v);
        }
        if (threadIdx.x < ST_COUNT && sh_stat[threadIdx.x]) {
            if (threadIdx.x == ST_MAX_CELLS || threadIdx.x == ST_MAX_EXTENT) atomicMax(&stats[threadIdx.x], sh_stat[threadIdx.x]);
            else atomicAdd(&stats[threadIdx.x], sh_stat[threadIdx.x]);
        }
    }
}

// ---------------------------------------------------------------- exclusive scan (3 kernels)
// in: n uint32 counts -> out: n+1 uint64 exclusive prefix (out[n] = total);
// second output: items per tile = ceil(count/chunk), scanned the same way.
constexpr int SCAN_BLOCK = 1024;

// work items of bin i: a tile's items are counted at its first bin (the chunks run over both
// classes of the tile together), its other bins count none
__device__ __forceinline__ unsigned long long bin_items(const unsigned int* counts, long long i, long long n,
                                                        unsigned int chunk) {
    if (i >= n || i % N_CLASSES != 0) return 0ull;
    unsigned long long c = 0;
#pragma unroll
    for (int k = 0; k < N_CLASSES; ++k) c += counts[i + k];
    return (c + chunk - 1) / chunk;
}

__global__ void __launch_bounds__(SCAN_BLOCK) k_scan_partials(const unsigned int* counts, long long n,
                                                              unsigned int chunk,
                                                              unsigned long long* part_pairs,
                                                              unsigned long long* part_items) {
    __shared__ unsigned long long sp[32], si[32];
    long long i = blockIdx.x * (long long)SCAN_BLOCK + threadIdx.x;
    unsigned long long c = i < n ? counts[i] : 0ull;
    unsigned long long it = bin_items(counts, i, n, chunk);
    for (int o = 16; o; o >>= 1) {
        c += __shfl_down_sync(0xffffffffu, c, o);
        it += __shfl_down_sync(0xffffffffu, it, o);
    }
    if ((threadIdx.x & 31) == 0) { sp[threadIdx.x >> 5] = c; si[threadIdx.x >> 5] = it; }
    __syncthreads();
    if (threadIdx.x < 32) {
        c = sp[threadIdx.x]; it = si[threadIdx.x];
        for (int o = 16; o; o >>= 1) {
            c += __shfl_down_sync(0xffffffffu, c, o);
            it += __shfl_down_sync(0xffffffffu, it, o);
        }
        if (threadIdx.x == 0) { part_pairs[blockIdx.x] = c; part_items[blockIdx.x] = it; }
    }
}

// single block: exclusive scan of the per-block partials in place; totals to totals[0..1]
__global__ void __launch_bounds__(SCAN_BLOCK) k_scan_top(unsigned long long* part_pairs,
                                                         unsigned long long* part_items, int nparts,
                                                         unsigned long long* totals) {
    __shared__ unsigned long long wp[32], wi[32];
    __shared__ unsigned long long carry[2];
    if (threadIdx.x == 0) { carry[0] = 0; carry[1] = 0; }
    __syncthreads();
    for (int base = 0; base < nparts; base += SCAN_BLOCK) {
        int i = base + threadIdx.x;
        unsigned long long a = i < nparts ? part_pairs[i] : 0ull, b = i < nparts ? part_items[i] : 0ull;
        unsigned long long ia = a, ib = b;
        int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
        for (int o = 1; o < 32; o <<= 1) {
            unsigned long long ta = __shfl_up_sync(0xffffffffu, ia, o), tb = __shfl_up_sync(0xffffffffu, ib, o);
            if (lane >= o) { ia += ta; ib += tb; }
        }
        if (lane == 31) { wp[w] = ia; wi[w] = ib; }
        __syncthreads();
        if (w == 0) {
            unsigned long long xa = wp[lane], xb = wi[lane];
            for (int o = 1; o < 32; o <<= 1) {
                unsigned long long ta = __shfl_up_sync(0xffffffffu, xa, o), tb = __shfl_up_sync(0xffffffffu, xb, o);
                if (lane >= o) { xa += ta; xb += tb; }
            }
            wp[lane] = xa; wi[lane] = xb;
        }
        __syncthreads();
        unsigned long long offa = carry[0] + (w ? wp[w - 1] : 0ull), offb = carry[1] + (w ? wi[w - 1] : 0ull);
        if (i < nparts) { part_pairs[i] = offa + ia - a; part_items[i] = offb + ib - b; }
        __syncthreads();
        if (threadIdx.x == SCAN_BLOCK - 1) { carry[0] = offa + ia; carry[1] = offb + ib; }
        __syncthreads();
    }
    if (threadIdx.x == 0) { totals[0] = carry[0]; totals[1] = carry[1]; }
}

__global__ void __launch_bounds__(SCAN_BLOCK) k_scan_final(const unsigned int* counts, long long n,
                                                           unsigned int chunk,
                                                           const unsigned long long* part_pairs,
                                                           const unsigned long long* part_items,
                                                           unsigned long long* tile_offsets,
                                                           unsigned long long* item_offsets) {
    __shared__ unsigned long long wp[32], wi[32];
    long long i = blockIdx.x * (long long)SCAN_BLOCK + threadIdx.x;
    unsigned long long a = i < n ? counts[i] : 0ull;
    unsigned long long b = bin_items(counts, i, n, chunk);
    unsigned long long ia = a, ib = b;
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int o = 1; o < 32; o <<= 1) {
        unsigned long long ta = __shfl_up_sync(0xffffffffu, ia, o), tb = __shfl_up_sync(0xffffffffu, ib, o);
        if (lane >= o) { ia += ta; ib += tb; }
    }
    if (lane == 31) { wp[w] = ia; wi[w] = ib; }
    __syncthreads();
    if (w == 0) {
        unsigned long long xa = wp[lane], xb = wi[lane];
        for (int o = 1; o < 32; o <<= 1) {
            unsigned long long ta = __shfl_up_sync(0xffffffffu, xa, o), tb = __shfl_up_sync(0xffffffffu, xb, o);
            if (lane >= o) { xa += ta; xb += tb; }
        }
        wp[lane] = xa; wi[lane] = xb;
    }
    __syncthreads();
    unsigned long long offa = part_pairs[blockIdx.x] + (w ? wp[w - 1] : 0ull);
    unsigned long long offb = part_items[blockIdx.x] + (w ? wi[w - 1] : 0ull);
    if (i < n) { tile_offsets[i] = offa + ia - a; item_offsets[i] = offb + ib - b; }
    if (i == n - 1) { tile_offsets[n] = offa + ia; item_offsets[n] = offb + ib; }
}

// work items: each tile's pair list cut into chunks
__global__ void k_items(const unsigned int* counts, long long n, unsigned int chunk,
                        const unsigned long long* tile_offsets,
                        const unsigned long long* item_offsets, Item* items) {
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;  // tile; n = number of tiles
    if (t >= n) return;
    unsigned int c = 0;
#pragma unroll
    for (int k = 0; k < N_CLASSES; ++k) c += counts[t * N_CLASSES + k];
    unsigned long long io = item_offsets[t * N_CLASSES], po = tile_offsets[t * N_CLASSES];
    for (unsigned int done = 0; done < c; done += chunk) {
        Item it;
        it.tile = (unsigned int)t;
        it.count = min(chunk, c - done);
        it.begin = po + done;
        items[io++] = it;
    }
}

// first work item whose pair list starts at or after s * step pairs, s = 0..ns-1 (the items ascend
// by `begin`): out[2s] = item index, out[2s+1] = its first pair (n_pairs past the end)
__global__ void k_slab_bounds(const Item* items, unsigned long long n_items, unsigned long long n_pairs,
                              unsigned long long step, int ns, unsigned long long* out) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= ns) return;
    const unsigned long long target = (unsigned long long)s * step;
    unsigned long long lo = 0, hi = n_items;  // first index with begin >= target
    while (lo < hi) {
        const unsigned long long mid = (lo + hi) >> 1;
        if (items[mid].begin >= target) hi = mid; else lo = mid + 1;
    }
    out[2 * s] = lo;
    out[2 * s + 1] = lo < n_items ? items[lo].begin : n_pairs;
}

// ---------------------------------------------------------------- a4-a6 binned deposit
struct DepositArgs {
    Particles part;
    Space space;
    const unsigned int* pair_ids;
    const Item* items;
    double mass_per_tet;
    int weight_mode;  // 0 mass, 1 signed volume
    int chord_axis;   // -1 adaptive, else 0..2
    unsigned long long* stats;
    double acc_scale, acc_inv_scale;  // fixed-point tile accumulators (PSD_ACC_FIXED): a power of two and its inverse
    // pair records (k_pair_records -> k_deposit_tiles), 18 doubles (144 bytes) each, one after the
    // other (a pair's data sits in two cache lines: the jobs of a slot read it through L1):
    //   [0..11] tile-local vertex coordinates (vertex v, axis x at 3 v + x), [12] weight (or the
    //   value of a "special" add), [13..16] the four faces' row words (u64), [17] word | cnts << 32.
    // rec_g == nullptr: the deposit kernel runs stage A itself (fused mode)
    const double* rec_g;
    unsigned long long rec_pair_begin;  // first pair (position in pair_ids) of the record buffer
    const void* tet_info;               // shared faces (psd_faces.cuh): the per-tet table, TetInfo[n_levels][6 N^3]
};

constexpr int REC_DOUBLES = 18;
__device__ __forceinline__ double rec_d(const DepositArgs& A, long long r, int c) { return __ldg(A.rec_g + r * REC_DOUBLES + c); }
__device__ __forceinline__ unsigned long long rec_rows(const DepositArgs& A, long long r, int f) {
    return __ldg(reinterpret_cast<const unsigned long long*>(A.rec_g) + r * REC_DOUBLES + 13 + f);
}
__device__ __forceinline__ unsigned int rec_word(const DepositArgs& A, long long r) {
    return __ldg(reinterpret_cast<const unsigned int*>(A.rec_g) + r * (2 * REC_DOUBLES) + 34);
}
__device__ __forceinline__ unsigned int rec_cnts(const DepositArgs& A, long long r) {
    return __ldg(reinterpret_cast<const unsigned int*>(A.rec_g) + r * (2 * REC_DOUBLES) + 35);
}



// a6, the tile accumulator.  Shared memory has no native 64-bit atomic add on sm_100a (fp64 and
// u64 atomicAdd both compile to an ATOMS.CAST.SPIN.64 compare-and-swap loop); only the 32-bit
// integer ATOMS.ADD is native.  With PSD_ACC_FIXED a cell is a 64-bit two's-complement fixed-point
// number (unit 1 / acc_scale, a power of two, so that the scaling is exact) held in two 32-bit
// limbs: the low limb is added with one native atomic that returns the old value, the carry out
// of it goes with the high limb in a second one.  Integer addition commutes and every carry is
// added exactly once, so the two limbs end up exact whatever the interleaving; sums wrap modulo
// 2^64, which is harmless as long as the final value of the cell fits (it is bounded by the
// chunk size times the mass of a tet, and acc_scale is chosen from that).
#ifndef PSD_ACC_FIXED
#define PSD_ACC_FIXED 1
#endif
struct TileShare {
#if PSD_ACC_FIXED
    unsigned int lo, hi;
#else
    double x;
#endif
};
__device__ __forceinline__ TileShare tile_share(double x, double scale) {
    TileShare q;
#if PSD_ACC_FIXED
    double y = x * scale;
    if (fabs(y) >= 0x1p62) y -= 0x1p64 * rint(y * 0x1p-64);  // sliver tets: reduce modulo 2^64 (exact)
    const long long v = __double2ll_rn(y);
    q.lo = (unsigned int)v; q.hi = (unsigned int)(v >> 32);
#else
    q.x = x;
#endif
    return q;
}
// The two limbs of cell i are at words i and 512 + i of the tile (not next to each other: the
// cells of the lanes of a warp then spread over all 32 banks).
__device__ __forceinline__ void tile_add(double* acc, int i, TileShare q) {
#if PSD_ACC_FIXED
    unsigned int* a = reinterpret_cast<unsigned int*>(acc) + i;
    const unsigned int old = atomicAdd(a, q.lo);
    atomicAdd(a + TILE_CELLS, q.hi + (unsigned int)(old + q.lo < old));
#else
    atomicAdd(acc + i, q.x);
#endif
}
__device__ __forceinline__ double tile_value(const double* acc, int i, double inv_scale) {
#if PSD_ACC_FIXED
    const unsigned int* a = reinterpret_cast<const unsigned int*>(acc);
    return (double)(long long)(((unsigned long long)a[TILE_CELLS + i] << 32) | a[i]) * inv_scale;
#else
    return acc[i];
#endif
}

#ifndef DEP_MIN_CTAS
#define DEP_MIN_CTAS 4
#endif
#ifndef DEP_WARPS_N
#define DEP_WARPS_N 4
#endif
constexpr int DEP_WARPS = DEP_WARPS_N;
constexpr int DEP_THREADS = DEP_WARPS * 32;
// per-warp scratch in doubles: tet slots [13][32] (12 tile-local coordinates + weight), polygon
// [3*LB_SLOTS][32], per-face row ranges [4][32] (u64), slot words [32] (u32)
constexpr int WARP_SCRATCH = (13 + 3 * LB_SLOTS) * 32 + 4 * 32 + 16;
constexpr int DEP_SMEM_BYTES = (TILE_CELLS + DEP_WARPS * WARP_SCRATCH) * 8;
// the records-only kernel (k_deposit_tiles<COUNT, true>) reads the slots' data straight from the
// pair records (L1): its per-warp scratch is the polygon buffer alone -> 6 CTAs per SM instead of 4
constexpr int WARP_SCRATCH_REC = 3 * LB_SLOTS * 32;
constexpr int DEP_SMEM_BYTES_REC = (TILE_CELLS + DEP_WARPS * WARP_SCRATCH_REC) * 8;
#ifndef DEP_MIN_CTAS_REC
#define DEP_MIN_CTAS_REC 6
#endif

// The general convex clip (clip_wall) of one face job, for the jobs the straight-line clip
// reports as ambiguous (lattice-aligned input): kept out of line, it runs rarely.
__device__ __noinline__ FaceClip face_clip_general(double* lane_poly) {  // triangle in slots 0..2
    PolyBuf<32> q{lane_poly};
    return face_clip<32, false>(q);
}

__device__ __forceinline__ void tile_geometry(const Space& s, unsigned int tile, int& level,
                                              int org[3], double*& out, long long str[3]) {
    if (!s.patch_mode) {
        int tz = tile % s.nt, ty = (tile / s.nt) % s.nt, tx = tile / (s.nt * s.nt);
        level = 0;
        org[0] = tx * TILE; org[1] = ty * TILE; org[2] = tz * TILE;
        str[0] = (long long)s.G * s.G; str[1] = s.G; str[2] = 1;
        out = s.out + org[0] * str[0] + org[1] * str[1] + org[2];
    } else {
        int tp3 = s.tp * s.tp * s.tp;
        unsigned int pi = tile / tp3, sub = tile % tp3;
        PatchDev pd = s.patches[pi];
        int sz = sub % s.tp, sy = (sub / s.tp) % s.tp, sx = sub / (s.tp * s.tp);
        level = pd.level;
        org[0] = pd.ox * s.P + sx * TILE; org[1] = pd.oy * s.P + sy * TILE; org[2] = pd.oz * s.P + sz * TILE;
        str[0] = (long long)s.P * s.P; str[1] = s.P; str[2] = 1;
        out = s.out + (long long)pi * s.P * s.P * s.P + (sx * TILE) * str[0] + (sy * TILE) * str[1] + sz * TILE;
    }
}

// ---------------------------------------------------------------- a1-a3 per pair: stage A
// One (tet, tile) pair, one periodic image of the tile: the tet rebuilt from its id (a1), its
// determinant and weight, tile-local vertices, chord axis, and per face the columns each row of
// its rectangle really meets.  Written to the lane's column of three [.][32] blocks:
//   wt [13][32] doubles  vertex v, coordinate x at row 3 v + x; weight at row 12
//   wr [4][32]  u64      per face: first row (3 bits), then 7 bits per row: first column, columns
//   ww [32]     u32      chord axis (2 bits), first / last cell of the tet along it in the tile
// A tet that goes to one cell whole (inside one cell, or degenerate) is returned as a "special" add.
//
// a4 in this formulation is the classification of (face, column) jobs: which columns of a row of
// the face's rectangle the triangle really meets (face_rows).  It runs in fp64 with a 1e-9 margin,
// or in fp32 with a margin that covers fp32's rounding ("fp32 classification
// with a conservative margin, fp64 clip for the survivors"): either way the set of jobs contains
// every column with a non-empty polygon, a job too many clips to nothing, so the deposit is the same.
template <typename T> struct RowNum;
template <> struct RowNum<double> {
    static constexpr bool exact_rect = true;
    static __device__ __forceinline__ int fl(double x) { return __double2int_rd(x); }
    static __device__ __forceinline__ int ce(double x) { return __double2int_ru(x); }
    static __device__ __forceinline__ double rcp(double x) { return fast_rcp(x); }
    static __device__ __forceinline__ double mad(double a, double b, double c) { return fma(a, b, c); }
};
template <> struct RowNum<float> {
    static constexpr bool exact_rect = false;
    static __device__ __forceinline__ int fl(float x) { return __float2int_rd(x); }
    static __device__ __forceinline__ int ce(float x) { return __float2int_ru(x); }
    static __device__ __forceinline__ float rcp(float x) {
        float r;
        asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
        return r;
    }
    static __device__ __forceinline__ float mad(float a, float b, float c) { return fmaf(a, b, c); }
};

// The row words of a tet's four faces (first row in bits 0..2, then 7 bits per row: first column
// (3), columns (4)) and the faces' job counts (8 bits each).  pu/pv/pw: the 4 vertices, tile-local;
// [lov,hiv] x [low,hiw]: the tet's cell range in the tile across the chord axis, lou: its first
// cell along it.  The w-extremes of (triangle n row strip) are at vertices inside the strip or
// where an edge crosses one of the strip's two lines.
//   T = double: rectangles exact, rows / columns with a margin of 1e-9 (a point that close to a
//       lattice line counts for both sides).
//   T = float:  with a = max |coordinate|, every rounded coordinate and difference is within
//       2^-23 a of its value, so e0 = 2^-19 a covers the row a vertex is in; a crossing point
//       w = w_i - (v_i - L) dw/dv is within 2^-23 a (3 |dw/dv| + 5) of its value when |dv| > e0 / 2
//       (then dv is known to 25 %), and when |dv| <= e0 / 2 both ends of the edge are within e0 of
//       the line, count for both rows, and the crossing lies between them; a crossing that the
//       rounded signs miss is within |dw/dv| 2^-23 a of a vertex that counts for both rows.  So
//       em = e0 (1 + max |dw/dv| over the tet's edges) covers every column decision.
template <typename T>
__device__ __forceinline__ unsigned int face_rows(const double pu[4], const double pv[4], const double pw[4],
                                                  const int lov, const int hiv, const int low, const int hiw,
                                                  const int lou, unsigned long long rows4[4]) {
    using R = RowNum<T>;
    T pvv[4], pww[4];
    T e0, em, er, erw;  // margins: row of a vertex, column of a point, rectangle rows, rectangle columns
    T slope[6];         // dw/dv of the 6 edges (i < j), index i + j - (i == 0 ? 1 : 0): 01 02 03 12 13 23
#pragma unroll
    for (int v = 0; v < 4; ++v) { pvv[v] = (T)pv[v]; pww[v] = (T)pw[v]; }
    T smax = (T)0;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = i + 1; j < 4; ++j) {
            const T dvv = pvv[j] - pvv[i];
            const T sl = (pww[j] - pww[i]) * R::rcp(dvv == (T)0 ? (T)1 : dvv);
            slope[i + j - (i == 0 ? 1 : 0)] = sl;
            if (!R::exact_rect) smax = fmax(smax, fabs(sl));
        }
    T puu[4];
    if (R::exact_rect) {
        e0 = (T)1e-9; em = (T)1e-9; er = (T)0; erw = (T)0;
#pragma unroll
        for (int v = 0; v < 4; ++v) puu[v] = (T)pu[v];
    } else {
        T amax = (T)1;
#pragma unroll
        for (int v = 0; v < 4; ++v) {
            puu[v] = (T)pu[v];
            amax = fmax(amax, fmax(fabs(puu[v]), fmax(fabs(pvv[v]), fabs(pww[v]))));
        }
        e0 = amax * (T)0x1p-19;
        em = R::mad(e0, smax, e0);
        er = e0; erw = em;
    }
    // per vertex: floor / ceil of (v, w) and ceil of u for the faces' rectangles (integer min / max:
    // floor and ceil are monotone); rows / columns the vertex belongs to with the margin
    int fv[4], cvv[4], fw[4], cww[4], cuu[4], rlo[4], rhi[4], klo[4], khi[4];
#pragma unroll
    for (int v = 0; v < 4; ++v) {
        rlo[v] = R::fl(pvv[v] - e0); rhi[v] = R::fl(pvv[v] + e0);
        klo[v] = R::fl(pww[v] - em); khi[v] = R::fl(pww[v] + em);
        if (R::exact_rect) {
            fv[v] = R::fl(pvv[v]); fw[v] = R::fl(pww[v]);
        } else {
            fv[v] = rlo[v]; fw[v] = klo[v];
        }
        cvv[v] = R::ce(pvv[v] + er); cww[v] = R::ce(pww[v] + erw);
        cuu[v] = R::ce(puu[v] + er);
    }
    // columns met by the face's three edges on the lattice line v = L (with the margin)
    auto line_cols = [&](const int a, const int b, const int d, const int L, int& clo, int& chi) {
        clo = 99; chi = -99;
        const int e0i[3] = {a, b, a}, e1i[3] = {b, d, d};   // edges with i < j: (a,b) (b,d) (a,d)
#pragma unroll
        for (int e = 0; e < 3; ++e) {
            const int i = e0i[e], j = e1i[e];
            const T di = pvv[i] - (T)L, dj = pvv[j] - (T)L;
            if (di * dj < (T)0) {
                const T w = R::mad(-di, slope[i + j - (i == 0 ? 1 : 0)], pww[i]);
                clo = min(clo, R::fl(w - em));
                chi = max(chi, R::fl(w + em));
            }
        }
    };
    unsigned int cnts = 0u;
#pragma unroll
    for (int f = 0; f < 4; ++f) {  // face f = the 3 vertices other than f
        const int a = f == 0 ? 1 : 0, b = f <= 1 ? 2 : 1, d = f == 3 ? 2 : 3;   // a < b < d
        // columns cv with minv < cv+1 and maxv > cv, inside the tet's tile range
        const int v0 = max(min(min(fv[a], fv[b]), fv[d]), lov);
        const int v1 = min(max(max(cvv[a], cvv[b]), cvv[d]) - 1, hiv);
        const int w0 = max(min(min(fw[a], fw[b]), fw[d]), low);
        const int w1 = min(max(max(cww[a], cww[b]), cww[d]) - 1, hiw);
        int c = 0;
        unsigned long long rows = 0ull;
        if (v1 >= v0 && w1 >= w0 && max(max(cuu[a], cuu[b]), cuu[d]) > lou) {
            rows = (unsigned long long)v0;
            int llo, lhi;
            line_cols(a, b, d, v0, llo, lhi);
#pragma unroll 1
            for (int r = v0; r <= v1; ++r) {
                int ulo, uhi;
                line_cols(a, b, d, r + 1, ulo, uhi);
                int rl = min(llo, ulo), rh = max(lhi, uhi);
                if (rlo[a] <= r && r <= rhi[a]) { rl = min(rl, klo[a]); rh = max(rh, khi[a]); }
                if (rlo[b] <= r && r <= rhi[b]) { rl = min(rl, klo[b]); rh = max(rh, khi[b]); }
                if (rlo[d] <= r && r <= rhi[d]) { rl = min(rl, klo[d]); rh = max(rh, khi[d]); }
                const int c0 = max(rl, w0), c1 = min(rh, w1);
                const int n = max(c1 - c0 + 1, 0);
                rows |= (unsigned long long)(n ? (c0 | n << 3) : 0) << (3 + 7 * (r - v0));
                c += n;
                llo = ulo; lhi = uhi;
            }
        }
        cnts |= (unsigned int)c << (8 * f);
        rows4[f] = rows;
    }
    return cnts;
}

// Rows of the fp64 classification that the other one does not cover (a check: must be 0).  Both
// words: first row in bits 0..2, then 7 bits per row (first column, columns).
__device__ __forceinline__ unsigned int rows_missed(const unsigned long long wide, const unsigned long long ref) {
    const int v0w = (int)(wide & 7ull), v0r = (int)(ref & 7ull);
    unsigned int missed = 0;
#pragma unroll 1
    for (int i = 0; i < TILE; ++i) {
        const unsigned int fr = (unsigned int)(ref >> (3 + 7 * i)) & 127u;
        const int n = (int)(fr >> 3);
        if (n == 0) continue;
        const int c0 = (int)(fr & 7u), k = v0r + i - v0w;
        const unsigned int fw = (k >= 0 && k < TILE) ? (unsigned int)(wide >> (3 + 7 * k)) & 127u : 0u;
        const int c0w = (int)(fw & 7u), nw = (int)(fw >> 3);
        missed += !(nw > 0 && c0w <= c0 && c0w + nw >= c0 + n);
    }
    return missed;
}

struct StageA {
    unsigned int missed; // ROWS = 2: rows of the fp64 classification not covered by the fp32 one
    unsigned int cnts;   // face jobs, 8 bits per face
    int my_images;       // periodic images of the tile this tet's range meets
    bool special;
    int special_cell;    // cell of the tile, (x*8+y)*8+z
    double special_val;
};
template <int SS, int ROWS>  // SS: stride of the [.][32] blocks in elements (32; 33 where they are read
                             // transposed); ROWS: 0 the rows in fp64, 1 in fp32, 2 in fp32 and checked
                             // against fp64 (face_rows)
__device__ __forceinline__ StageA stage_a(const DepositArgs& A, const bool have, const unsigned int id, const int img,
                                          const int org[3], const int Gl, const double scale, double* wt,
                                          unsigned long long* wr, unsigned int* ww) {
    StageA o;
    o.cnts = 0u; o.my_images = 0; o.special = false; o.special_cell = 0; o.special_val = 0.0; o.missed = 0u;
            Tet t;
            double det = 1.0;
            int nimg[3] = {1, 1, 1}, mlo[3] = {0, 0, 0};
            if (have) {
                double P[4][3];
                load_tet_vertices(A.part, id / 6, id % 6, P);
                finish_tet(P, scale, t);
                det = tet_det(t.g);
#pragma unroll
                for (int x = 0; x < 3; ++x) {  // periodic images of this tile met by the tet's range
                    mlo[x] = -floor_div(org[x] + TILE - 1 - t.lo[x], Gl);
                    nimg[x] = floor_div(t.hi[x] - org[x], Gl) - mlo[x] + 1;
                }
                o.my_images = nimg[0] * nimg[1] * nimg[2];
            }
            if (img < o.my_images) {
                int m[3] = {mlo[0] + img % nimg[0], mlo[1] + (img / nimg[0]) % nimg[1],
                            mlo[2] + img / (nimg[0] * nimg[1])};
                int lo[3], hi[3];
                double gl[4][3];
#pragma unroll
                for (int x = 0; x < 3; ++x) {
                    int o = org[x] + m[x] * Gl;
                    lo[x] = max(t.lo[x] - o, 0);
                    hi[x] = min(t.hi[x] - o, TILE - 1);
#pragma unroll
                    for (int v = 0; v < 4; ++v) {
                        gl[v][x] = t.g[v][x] - (double)o;
                        wt[(3 * v + x) * SS] = gl[v][x];
                    }
                }
                wt[12 * SS] = A.weight_mode == 0 ? (det != 0.0 ? 6.0 * A.mass_per_tet / det : 0.0) : 1.0;
                int ax = A.chord_axis;
                if (ax < 0) {  // longest extent inside the tile -> fewest, longest columns
                    int e0 = hi[0] - lo[0], e1 = hi[1] - lo[1], e2 = hi[2] - lo[2];
                    ax = (e0 >= e1 && e0 >= e2) ? 0 : (e1 >= e2 ? 1 : 2);
                }
                const int av = (ax + 1) % 3, aw = (ax + 2) % 3;
                bool rect_written = false;
                if (det == 0.0) {  // degenerate: whole mass to the centroid cell (Q6)
                    if (A.weight_mode == 0) {
                        int c[3];
                        bool in = true;
#pragma unroll
                        for (int x = 0; x < 3; ++x) {
                            double cen = (t.g[0][x] + t.g[1][x] + t.g[2][x] + t.g[3][x]) / 4.0;
                            c[x] = __double2int_rd(cen) - (org[x] + m[x] * Gl);
                            in = in && c[x] >= 0 && c[x] < TILE;
                        }
                        if (in) { o.special = true; o.special_cell = (c[0] * TILE + c[1]) * TILE + c[2]; o.special_val = A.mass_per_tet; }
                    }
                } else if (t.lo[0] == t.hi[0] && t.lo[1] == t.hi[1] && t.lo[2] == t.hi[2]) {
                    // a4, tet inside one cell ("trivial cases"): the whole tet goes
                    // to that cell -- m, or its signed volume det/6 in signed-volume mode
                    o.special = true; o.special_cell = (lo[0] * TILE + lo[1]) * TILE + lo[2];
                    o.special_val = A.weight_mode == 0 ? A.mass_per_tet : det * (1.0 / 6.0);
                } else {
                    // per face the columns each row of its rectangle meets (row words + job counts),
                    // in fp64 with a 1e-9 margin, or (F32) in fp32 with a margin that covers its rounding
                    double pu4[4], pv4[4], pw4[4];
#pragma unroll
                    for (int v = 0; v < 4; ++v) {  // read back through the runtime axis (the lane's own stores above)
                        pu4[v] = wt[(3 * v + ax) * SS]; pv4[v] = wt[(3 * v + av) * SS]; pw4[v] = wt[(3 * v + aw) * SS];
                    }
                    const int lov = av == 0 ? lo[0] : (av == 1 ? lo[1] : lo[2]);
                    const int hiv = av == 0 ? hi[0] : (av == 1 ? hi[1] : hi[2]);
                    const int low = aw == 0 ? lo[0] : (aw == 1 ? lo[1] : lo[2]);
                    const int hiw = aw == 0 ? hi[0] : (aw == 1 ? hi[1] : hi[2]);
                    const int lou = ax == 0 ? lo[0] : (ax == 1 ? lo[1] : lo[2]);
                    unsigned long long rows4[4];
                    if (ROWS) o.cnts = face_rows<float>(pu4, pv4, pw4, lov, hiv, low, hiw, lou, rows4);
                    else o.cnts = face_rows<double>(pu4, pv4, pw4, lov, hiv, low, hiw, lou, rows4);
                    if (ROWS == 2) {
                        unsigned long long ref4[4];
                        face_rows<double>(pu4, pv4, pw4, lov, hiv, low, hiw, lou, ref4);
#pragma unroll
                        for (int f = 0; f < 4; ++f) o.missed += rows_missed(rows4[f], ref4[f]);
                    }
#pragma unroll
                    for (int f = 0; f < 4; ++f) wr[f * SS] = rows4[f];
                    rect_written = true;
                }
                const int lou = ax == 0 ? lo[0] : (ax == 1 ? lo[1] : lo[2]);
                const int hiu = ax == 0 ? hi[0] : (ax == 1 ? hi[1] : hi[2]);
                if (!rect_written) { wr[0] = 0ull; wr[SS] = 0ull; wr[2 * SS] = 0ull; wr[3 * SS] = 0ull; }
                *ww = (unsigned int)(ax | lou << 2 | hiu << 5);
            }
    return o;
}

// The pair records of a range of work items: stage A of every pair (image 0), one thread per pair,
// written record by record (18 doubles each; the deposit kernel's jobs read a slot's record through L1).  Splitting stage A off keeps the deposit kernel's instruction footprint inside
// the 32 KB instruction cache (with stage A inlined 18 % of its stall samples were no-instruction).
// Record index = (pair's position in the item, taken from the item's end) + item.begin - rec_pair_begin.
constexpr int REC_THREADS = 128;
#ifndef REC_MIN_CTAS
#define REC_MIN_CTAS 6
#endif
template <int ROWS>
__global__ void __launch_bounds__(REC_THREADS, REC_MIN_CTAS) k_pair_records(DepositArgs A) {
    // per warp: the 32 records field by field, [18][32] 8-byte words (rows 0..12 doubles, 13..16 the
    // row words, 17 word | cnts << 32), written out as one contiguous block of 32 x 18 words
    constexpr int SS = 33;  // padded: the block is read transposed when it is written out
    __shared__ unsigned long long stg[REC_THREADS / 32][REC_DOUBLES * SS];
    __shared__ unsigned int sww[REC_THREADS / 32][32];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double* swt = reinterpret_cast<double*>(stg[warp]);
    unsigned long long* swr = stg[warp] + 13 * SS;
    const Item item = A.items[blockIdx.x];
    int level, org[3];
    double* out;
    long long str[3];
    tile_geometry(A.space, item.tile, level, org, out, str);
    const double scale = level_scale(A.space, level);
    const int Gl = level_G(A.space, level);
    for (unsigned int k0 = 0; k0 < item.count; k0 += REC_THREADS) {
        const unsigned int k = k0 + threadIdx.x;
        const bool have = k < item.count;
        const unsigned int id = have ? A.pair_ids[item.begin + (item.count - 1u - k)] : 0u;
        __syncwarp();
        const StageA sa = stage_a<SS, ROWS>(A, have, id, 0, org, Gl, scale, swt + lane, swr + lane, &sww[warp][lane]);
        if (ROWS == 2 && sa.missed) atomicAdd(&A.stats[ST_ROWS_MISSED], (unsigned long long)sa.missed);
        if (have) {
            if (sa.special) swt[12 * SS + lane] = sa.special_val;
            const unsigned int word = (sww[warp][lane] & 0xffu) | (unsigned int)sa.special << 8 |
                                      (unsigned int)sa.special_cell << 9 | (unsigned int)min(sa.my_images, 16383) << 18;
            stg[warp][17 * SS + lane] = (unsigned long long)word | (unsigned long long)sa.cnts << 32;
        }
        __syncwarp();
        // the warp's records (k0 + 32 warp .. + 31, those that exist) as one coalesced block
        const unsigned int kw = k0 + 32u * warp;
        if (kw < item.count) {
            const int valid = (int)min(32u, item.count - kw);
            unsigned long long* dst = reinterpret_cast<unsigned long long*>(const_cast<double*>(A.rec_g)) +
                                      ((long long)(item.begin - A.rec_pair_begin) + kw) * REC_DOUBLES;
#pragma unroll
            for (int q = 0; q < REC_DOUBLES; ++q) {
                const int d = q * 32 + lane;
                const int j = (d * 3641) >> 16;  // d / 18 for d < 576
                const int c = d - j * REC_DOUBLES;
                if (j < valid) dst[d] = stg[warp][c * SS + j];
            }
        }
    }
}

// One CTA per work item (a chunk of one tile's pair list), an 8^3 fp64 accumulator in shared
// memory.  Each warp takes 32 pairs at a time:
//   stage A  lane = pair: build the tet (a1), its determinant and weight, tile-local vertices
//            into the warp's slots; per face the rectangle of columns its projection meets.
//   stage B  the face jobs (slot, face, column) of the 32 slots, face by face, are numbered by a
//            warp prefix sum of the rectangle sizes, 32 at a time with lane = job: the triangle
//            against its column in straight-line code (tri_square_clip: parametric clip of the 3
//            edges, corners by wall ids; no vertex list is edited, so the lanes do not diverge on
//            the number of walls), projected area and moment, trivial cells.
//   stage C  the cutting planes of the 32 polygons re-numbered over the lanes, closed-form plane
//            integrals, shares added to the tile (a4-a6).
// The tile is flushed to global memory with fp64 reductions at the end (a6).
// REC = true: every pair has a record and meets its tile in one periodic image only (the host
// checks the largest cell range against the grid): no stage A code, no slot staging in shared memory.
template <bool COUNT, bool REC>
__global__ void __launch_bounds__(DEP_THREADS, REC ? DEP_MIN_CTAS_REC : DEP_MIN_CTAS) k_deposit_tiles(DepositArgs A) {
    extern __shared__ double smem[];
    double* acc = smem;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double* wtet = smem + TILE_CELLS + warp * (REC ? WARP_SCRATCH_REC : WARP_SCRATCH);  // [13][32] (not REC)
    double* wpoly = REC ? wtet : wtet + 13 * 32;                                       // [3 * LB_SLOTS][32]
    unsigned long long* wrect = reinterpret_cast<unsigned long long*>(wpoly + 3 * LB_SLOTS * 32);  // [4][32] (not REC)
    unsigned int* wword = reinterpret_cast<unsigned int*>(wrect + 4 * 32);             // [32] (not REC)
    PolyBuf<32> poly{wpoly + lane};
    // slots 6..9 of the lane's polygon buffer hold the corners of the column's unit square: their
    // (v, w) never change (the general clip may overwrite slot 6: restored before the next job)
    poly.at(6, 1) = 0.0; poly.at(6, 2) = 0.0; poly.at(7, 1) = 1.0; poly.at(7, 2) = 0.0;
    poly.at(8, 1) = 1.0; poly.at(8, 2) = 1.0; poly.at(9, 1) = 0.0; poly.at(9, 2) = 1.0;
    bool slot6_dirty = false;

    const Item item = A.items[blockIdx.x];
    int level, org[3];
    double* out;
    long long str[3];
    tile_geometry(A.space, item.tile, level, org, out, str);
    const double scale = level_scale(A.space, level);
    const int Gl = level_G(A.space, level);

    __shared__ unsigned int sh_next;  // next batch of 32 pairs: warps fetch batches as they finish
    for (int i = threadIdx.x; i < TILE_CELLS; i += DEP_THREADS) acc[i] = 0.0;
    if (threadIdx.x == 0) sh_next = 0u;
    __syncthreads();

    JobCounters cnt = {0, 0, 0, 0, 0};

    for (;;) {
        unsigned int base = 0;
        if (lane == 0) base = atomicAdd(&sh_next, 32u);
        base = __shfl_sync(0xffffffffu, base, 0);
        if (base >= item.count) break;
        // ---- a1: each lane builds one tet of the batch.  The tet is rebuilt from its id for every
        // periodic image of the tile it meets (almost always one), so that nothing of stage A stays
        // in registers across stages B and C.
        const bool have = base + lane < item.count;
        // the list is taken from its end: the large class first, the small pairs last, so that the
        // warps of the CTA reach the end-of-item barrier closer together
        const unsigned int id = (!REC && have) ? A.pair_ids[item.begin + (item.count - 1u - (base + lane))] : 0u;
        // record of slot 0 of this batch (REC: the slots' data is read from the records where it is used)
        const long long rb = (long long)(item.begin - A.rec_pair_begin) + base;
        int max_images = 1;
        for (int img = 0; img < max_images; ++img) {
            // ---- stage A: slot = lane.  From the pair records (k_pair_records ran it for image 0), or
            // here: the further periodic images of a tile (tiny grids only), and the fused mode
            __syncwarp();
            StageA sa;
            if (REC) {
                sa.cnts = 0u; sa.my_images = 1; sa.special = false; sa.special_cell = 0; sa.special_val = 0.0;
                if (have) {
                    // the slot's record into L1 ahead of its jobs (its tail is read just below)
                    asm volatile("prefetch.global.L1 [%0];" ::"l"(A.rec_g + (rb + lane) * REC_DOUBLES));
                    const unsigned int word = rec_word(A, rb + lane);
                    sa.cnts = rec_cnts(A, rb + lane);
                    sa.special = (word >> 8) & 1u;
                    sa.special_cell = (int)((word >> 9) & 511u);
                    if (sa.special) sa.special_val = rec_d(A, rb + lane, 12);
                }
            } else if (A.rec_g != nullptr && img == 0) {
                sa.cnts = 0u; sa.my_images = 0; sa.special = false; sa.special_cell = 0; sa.special_val = 0.0;
                if (have) {
                    const long long r = (long long)(item.begin - A.rec_pair_begin) + (base + lane);
#pragma unroll
                    for (int c = 0; c < 13; ++c) wtet[c * 32 + lane] = rec_d(A, r, c);
#pragma unroll
                    for (int f = 0; f < 4; ++f) wrect[f * 32 + lane] = rec_rows(A, r, f);
                    const unsigned int word = rec_word(A, r);
                    wword[lane] = word & 0xffu;
                    sa.cnts = rec_cnts(A, r);
                    sa.special = (word >> 8) & 1u;
                    sa.special_cell = (int)((word >> 9) & 511u);
                    sa.special_val = wtet[12 * 32 + lane];
                    sa.my_images = (int)(word >> 18);
                }
            } else {
                sa = stage_a<32, 0>(A, have, id, img, org, Gl, scale, wtet + lane, wrect + lane, wword + lane);
            }
            if (sa.special) tile_add(acc, sa.special_cell, tile_share(sa.special_val, A.acc_scale));
            const unsigned int cnts = sa.cnts;
            if (!REC && img == 0) max_images = __reduce_max_sync(0xffffffffu, sa.my_images);
            // ---- stages B + C for 32 jobs (a lambda with a single call site: its code is large).
            // B: lane = face job (slot, f, cv, cw): clip, area and moment, trivial cells.  C: the
            // cutting planes (polygon, a) of the 32 jobs, numbered by a warp prefix sum, lane = plane;
            // the kept part above the plane is integrated in closed form; +R to cell a, -R to a-1.
            auto run_jobs = [&](const bool act, const int slot, const int f, const int cv, const int cw) {
                unsigned int f_order = 0, f_info = 0, f_floors = 0;
                int f_afirst = 0, k = 0;
                double f_w = 0.0;
                if (act) {
                    if (COUNT) cnt.jobs++;
                    const unsigned int word = REC ? rec_word(A, rb + slot) : wword[slot];
                    const int ax = word & 3, c_lo = (word >> 2) & 7, c_hi = (word >> 5) & 7;
                    const int av = ax == 2 ? 0 : ax + 1, aw = ax == 0 ? 2 : ax - 1;
                    // the face triangle, column-local
                    const double* ts = wtet + slot;
                    const long long rs = rb + slot;           // REC: the slot's record
                    const unsigned int fv = FACE_TABLE >> (6 * f);
                    const double ov = (double)cv, ow = (double)cw;
                    double U[3], V[3], W[3];
#pragma unroll
                    for (int i = 0; i < 3; ++i) {
                        const int vi = (fv >> (2 * i)) & 3;
                        if (REC) {
                            U[i] = rec_d(A, rs, 3 * vi + ax);
                            V[i] = rec_d(A, rs, 3 * vi + av) - ov;
                            W[i] = rec_d(A, rs, 3 * vi + aw) - ow;
                        } else {
                            U[i] = ts[(3 * vi + ax) * 32];
                            V[i] = ts[(3 * vi + av) * 32] - ov;
                            W[i] = ts[(3 * vi + aw) * 32] - ow;
                        }
                    }
                    f_w = REC ? rec_d(A, rs, 12) : ts[12 * 32];
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
                        if (lb.sign < 0) f_w = -f_w;  // clockwise triangle: the polygon is its mirror image
                    }
                    if (fc.n >= 3 && fc.ice > c_lo) {
                        if (COUNT) cnt.face_clips++;
                        const FaceRun fr = face_run(fc, c_lo, c_hi);
                        // strides of (u,v,w) in the 8^3 accumulator, index (x*8+y)*8+z
                        const int su = ax == 0 ? 64 : (ax == 1 ? 8 : 1);
                        const int sv = av == 0 ? 64 : (av == 1 ? 8 : 1);
                        const int sw = aw == 0 ? 64 : (aw == 1 ? 8 : 1);
                        const int colofs = cv * sv + cw * sw;
                        // trivial part: cells entirely below Q get its projected area, the cell
                        // holding umin gets M1 - c A
                        {
                            const int full_hi = min(fr.t_hi, fc.ifl - 1);  // cells entirely below Q
                            const double wA = f_w * fc.A;
                            if (wA != 0.0) {
                                const TileShare qA = tile_share(wA, A.acc_scale);
#pragma unroll
                                for (int cc = 0; cc < TILE; ++cc) {
                                    const int c = c_lo + cc;
                                    if (c > full_hi) break;
                                    tile_add(acc, colofs + c * su, qA);
                                    if (COUNT) cnt.cells++;
                                }
                            }
                            if (fr.t_hi >= fc.ifl && fc.ifl >= c_lo) {  // the cell holding umin
                                const double D = fma(-(double)fc.ifl, fc.A, fc.M1);
                                if (D != 0.0) {
                                    tile_add(acc, colofs + fc.ifl * su, tile_share(f_w * D, A.acc_scale));
                                    if (COUNT) cnt.cells++;
                                }
                            }
                        }
                        k = max(fr.a_last - fr.a_first + 1, 0);
                        f_order = fc.order;
                        f_floors = fc.floors;
                        f_afirst = fr.a_first;
                        f_info = (unsigned)colofs | (unsigned)ax << 9 | (unsigned)c_lo << 11 | (unsigned)c_hi << 14 |
                                 (unsigned)fc.n << 17 | fc.below0 << 20;
                    }
                }
                __syncwarp();
                int pre2 = k;
                for (int o = 1; o < 32; o <<= 1) {
                    int y = __shfl_up_sync(0xffffffffu, pre2, o);
                    if (lane >= o) pre2 += y;
                }
                const int total2 = __shfl_sync(0xffffffffu, pre2, 31);
                pre2 -= k;
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
                    const int s_afirst = __shfl_sync(0xffffffffu, f_afirst, src);
                    const double s_w = __shfl_sync(0xffffffffu, f_w, src);
                    if (e < total2) {
                        const int a = s_afirst + (e - s_pre);
                        const int colofs = s_info & 511, ax = (s_info >> 9) & 3;
                        const int c_lo = (s_info >> 11) & 7, c_hi = (s_info >> 14) & 7, n = (s_info >> 17) & 7;
                        const int su = ax == 0 ? 64 : (ax == 1 ? 8 : 1);
                        PolyBuf<32> qs{wpoly + src};
                        const double R = plane_integral6_mask<32>(qs, s_order, n, (double)a, plane_mask_from_floors(s_floors, (s_info >> 20) & 127u, n, a)) *
                                         (1.0 / 6.0) * s_w;
                        if (COUNT) cnt.plane_evals++;
                        if (R != 0.0) {
                            if (a <= c_hi) { tile_add(acc, colofs + a * su, tile_share(R, A.acc_scale)); if (COUNT) cnt.cells++; }
                            if (a - 1 >= c_lo) { tile_add(acc, colofs + (a - 1) * su, tile_share(-R, A.acc_scale)); if (COUNT) cnt.cells++; }
                        }
                    }
                }
                __syncwarp();
            };
            // ---- the face jobs (slot, face, row, column) of the 32 slots, numbered by ONE warp prefix
            // sum of the slots' job counts (all four faces together: one partly filled pass per batch,
            // not one per face); a loop with a single call site of run_jobs
            __syncwarp();
            const int njobs = (int)((cnts & 255u) + ((cnts >> 8) & 255u) + ((cnts >> 16) & 255u) + (cnts >> 24));
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
                int slot = 0;  // largest slot with pre[slot] <= job
#pragma unroll
                for (int step = 16; step; step >>= 1) {
                    int probe = __shfl_sync(0xffffffffu, pre, slot + step);
                    if (probe <= job) slot += step;
                }
                const int spre = __shfl_sync(0xffffffffu, pre, slot);
                const unsigned int scnt = __shfl_sync(0xffffffffu, cnts, slot);
                int cv = 0, cw = 0, f = 0;
                const bool act = job < total;
                if (act) {
                    // decode (face, row, column): the slot's four face counts, then bits 0..2 of the
                    // face's word = first row, then 7 bits per row = first column (3), columns (4)
                    int local = job - spre;
                    unsigned int sc = scnt;
#pragma unroll
                    for (int q = 0; q < 3; ++q) {
                        const int n = (int)(sc & 255u);
                        if (local < n) break;
                        local -= n; ++f; sc >>= 8;
                    }
                    unsigned long long rw = REC ? rec_rows(A, rb + slot, f) : wrect[f * 32 + slot];
                    cv = (int)(rw & 7ull);
                    rw >>= 3;
#pragma unroll
                    for (int r = 0; r < TILE; ++r) {
                        const int n = (int)(rw >> 3) & 15;
                        if (local < n) break;
                        local -= n; ++cv; rw >>= 7;
                    }
                    cw = ((int)rw & 7) + local;
                }
                run_jobs(act, slot, f, cv, cw);
            }
        }
    }
    __syncthreads();
    // ---- a6: flush the tile with fp64 reductions (other work items may hold the same tile)
    for (int i = threadIdx.x; i < TILE_CELLS; i += DEP_THREADS) {
        const double v = tile_value(acc, i, A.acc_inv_scale);
        if (v != 0.0) {
            int cz = i & 7, cy = (i >> 3) & 7, cx = i >> 6;
            atomicAdd(out + cx * str[0] + cy * str[1] + cz, v);
        }
    }
    if (COUNT) {
        unsigned int a = __reduce_add_sync(0xffffffffu, cnt.jobs), b = __reduce_add_sync(0xffffffffu, cnt.face_clips);
        unsigned int c = __reduce_add_sync(0xffffffffu, cnt.plane_evals), d = __reduce_add_sync(0xffffffffu, cnt.cells);
        if (lane == 0) {
            atomicAdd(&A.stats[ST_TASKS], (unsigned long long)a);
            atomicAdd(&A.stats[ST_FACE_CLIPS], (unsigned long long)b);
            atomicAdd(&A.stats[ST_PLANE_CLIPS], (unsigned long long)c);
            atomicAdd(&A.stats[ST_CELLS], (unsigned long long)d);
        }
        const unsigned int e = __reduce_add_sync(0xffffffffu, cnt.general);
        if (lane == 0 && e) atomicAdd(&A.stats[ST_GENERAL], (unsigned long long)e);
    }
}

// ---------------------------------------------------------------- direct path (any G)
// One thread per tet: all its face jobs (face, column) in ONE flattened loop (lanes of a warp run
// the same job body whatever face or column they are at), polygon and tet-local vertices in
// warp-interleaved shared memory, global fp64 reductions with periodic wrap.  The plain path:
// PSD_OPT_KERNEL = 1, and grids the tiling does not divide.
constexpr int DIR_THREADS = 128;
constexpr int DIR_WARP_SCRATCH = (12 + 3 * POLY_CAP) * 32;  // doubles per warp

template <bool COUNT>
__global__ void __launch_bounds__(DIR_THREADS) k_deposit_direct(DepositArgs A) {
    __shared__ double scratch[(DIR_THREADS / 32) * DIR_WARP_SCRATCH];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double* ts = scratch + warp * DIR_WARP_SCRATCH + lane;   // [12][32]: vertex v, coord x at (3v+x)*32
    PolyBuf<32> poly{ts + 12 * 32};
    const int64_t ntet = (int64_t)6 * A.part.N * A.part.N * A.part.N;
    int64_t id = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    JobCounters cnt = {0, 0, 0, 0, 0};
    if (id < ntet) {
        const Space& s = A.space;
        const int G = s.G;
        double P[4][3];
        load_tet_vertices(A.part, id / 6, (int)(id % 6), P);
        Tet t;
        finish_tet(P, level_scale(s, 0), t);
        double det = tet_det(t.g);
        if (det == 0.0) {
            if (A.weight_mode == 0) {
                int c[3];
#pragma unroll
                for (int x = 0; x < 3; ++x)
                    c[x] = wrap_mod(__double2int_rd((t.g[0][x] + t.g[1][x] + t.g[2][x] + t.g[3][x]) / 4.0), G);
                atomicAdd(&s.out[((long long)c[0] * G + c[1]) * G + c[2]], A.mass_per_tet);
            }
        } else if (t.lo[0] == t.hi[0] && t.lo[1] == t.hi[1] && t.lo[2] == t.hi[2]) {
            // a4, tet inside one cell: no clipping
            atomicAdd(&s.out[((long long)wrap_mod(t.lo[0], G) * G + wrap_mod(t.lo[1], G)) * G + wrap_mod(t.lo[2], G)],
                      A.weight_mode == 0 ? A.mass_per_tet : det * (1.0 / 6.0));
        } else {
            const double w = A.weight_mode == 0 ? 6.0 * A.mass_per_tet / det : 1.0;
            int ax = A.chord_axis;
            if (ax < 0) {
                int e0 = t.hi[0] - t.lo[0], e1 = t.hi[1] - t.lo[1], e2 = t.hi[2] - t.lo[2];
                ax = (e0 >= e1 && e0 >= e2) ? 0 : (e1 >= e2 ? 1 : 2);
            }
            const int av = ax == 2 ? 0 : ax + 1, aw = ax == 0 ? 2 : ax - 1;
            // coordinates local to the tet's first cell, in (u, v, w) order
            int lo_u = 0, lo_v = 0, lo_w = 0, nu = 0, nv = 0, nw = 0;
#pragma unroll
            for (int x = 0; x < 3; ++x) {
                const int role = x == ax ? 0 : (x == av ? 1 : 2);
                if (role == 0) { lo_u = t.lo[x]; nu = t.hi[x] - t.lo[x]; }
                if (role == 1) { lo_v = t.lo[x]; nv = t.hi[x] - t.lo[x]; }
                if (role == 2) { lo_w = t.lo[x]; nw = t.hi[x] - t.lo[x]; }
#pragma unroll
                for (int v = 0; v < 4; ++v) ts[(3 * v + role) * 32] = t.g[v][x] - (double)t.lo[x];
            }
            // per face: the rectangle of columns its projection meets (face f = vertices other than f)
            int rv0[4], rv1[4], rw0[4], rw1[4];
            {
                int fv[4], cvv[4], fw[4], cww[4];  // per-vertex floors / ceils; integer min / max per face
#pragma unroll
                for (int v = 0; v < 4; ++v) {
                    const double cv = ts[(3 * v + 1) * 32], cw = ts[(3 * v + 2) * 32];
                    fv[v] = __double2int_rd(cv); cvv[v] = __double2int_ru(cv);
                    fw[v] = __double2int_rd(cw); cww[v] = __double2int_ru(cw);
                }
#pragma unroll
                for (int f = 0; f < 4; ++f) {
                    const int a = f == 0 ? 1 : 0, b = f <= 1 ? 2 : 1, d = f == 3 ? 2 : 3;
                    rv0[f] = max(min(min(fv[a], fv[b]), fv[d]), 0); rv1[f] = min(max(max(cvv[a], cvv[b]), cvv[d]) - 1, nv);
                    rw0[f] = max(min(min(fw[a], fw[b]), fw[d]), 0); rw1[f] = min(max(max(cww[a], cww[b]), cww[d]) - 1, nw);
                    if (rv1[f] < rv0[f] || rw1[f] < rw0[f]) { rv1[f] = rv0[f] - 1; rw1[f] = rw0[f] - 1; }  // empty
                }
            }
            // periodic wrap without a division per cell: the first cell wrapped once, then steps
            const int wu0 = wrap_mod(lo_u, G), wv0 = wrap_mod(lo_v, G), ww0 = wrap_mod(lo_w, G);
            auto wrapped = [G](int first, int off) { int c = first + off; while (c >= G) c -= G; return c; };
            // strides of (u,v,w) in the grid, index (x*G+y)*G+z
            const long long su = ax == 0 ? (long long)G * G : (ax == 1 ? G : 1);
            const long long sv = av == 0 ? (long long)G * G : (av == 1 ? G : 1);
            const long long sw = aw == 0 ? (long long)G * G : (aw == 1 ? G : 1);
            // ---- the flattened job loop: state (f, cv, cw) advanced incrementally
            int f = -1, cv = 0, cw = 0, v1 = -1, w0 = 0, w1 = -1;
            for (;;) {
                ++cw;
                if (cw > w1) { cw = w0; ++cv; }
                while (cv > v1) {  // next non-empty face
                    ++f;
                    if (f >= 4) break;
                    const int a0 = f == 0 ? rv0[0] : (f == 1 ? rv0[1] : (f == 2 ? rv0[2] : rv0[3]));
                    v1 = f == 0 ? rv1[0] : (f == 1 ? rv1[1] : (f == 2 ? rv1[2] : rv1[3]));
                    w0 = f == 0 ? rw0[0] : (f == 1 ? rw0[1] : (f == 2 ? rw0[2] : rw0[3]));
                    w1 = f == 0 ? rw1[0] : (f == 1 ? rw1[1] : (f == 2 ? rw1[2] : rw1[3]));
                    cv = a0; cw = w0;
                }
                if (f >= 4) break;
                const unsigned int fv = FACE_TABLE >> (6 * f);
                const double ov = (double)cv, ow = (double)cw;
#pragma unroll
                for (int i = 0; i < 3; ++i) {
                    const int vi = (fv >> (2 * i)) & 3;
                    poly.at(i, 0) = ts[(3 * vi + 0) * 32];
                    poly.at(i, 1) = ts[(3 * vi + 1) * 32] - ov;
                    poly.at(i, 2) = ts[(3 * vi + 2) * 32] - ow;
                }
                double* col = s.out + wrapped(wv0, cv) * sv + wrapped(ww0, cw) * sw;
                face_job<32, COUNT>(poly, 0, nu, [&](int c, double D) {
                    atomicAdd(col + wrapped(wu0, c) * su, w * D);
                }, &cnt);
            }
        }
    }
    if (COUNT) {
        unsigned int a = __reduce_add_sync(0xffffffffu, cnt.jobs), b = __reduce_add_sync(0xffffffffu, cnt.face_clips);
        unsigned int c = __reduce_add_sync(0xffffffffu, cnt.plane_evals), d = __reduce_add_sync(0xffffffffu, cnt.cells);
        if ((threadIdx.x & 31) == 0) {
            atomicAdd(&A.stats[ST_TASKS], (unsigned long long)a);
            atomicAdd(&A.stats[ST_FACE_CLIPS], (unsigned long long)b);
            atomicAdd(&A.stats[ST_PLANE_CLIPS], (unsigned long long)c);
            atomicAdd(&A.stats[ST_CELLS], (unsigned long long)d);
        }
    }
}

// census-only statistics for the direct path (no tiles): sum/max cells, histogram, inverted.
// Per-block partial results in shared memory, one set of global atomics per block.
__global__ void __launch_bounds__(256) k_tet_stats(Particles p, double scale, unsigned long long* stats,
                                                   unsigned long long* hist) {
    __shared__ unsigned int sh_hist[64];
    __shared__ unsigned long long sh_stat[ST_COUNT];
    if (threadIdx.x < 64) sh_hist[threadIdx.x] = 0;
    if (threadIdx.x < ST_COUNT) sh_stat[threadIdx.x] = 0;
    __syncthreads();
    int64_t ntet = (int64_t)6 * p.N * p.N * p.N;
    int64_t id = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    unsigned long long nc = 0;
    unsigned int inv = 0, deg = 0, suspect = 0;
    if (id < ntet) {
        double P[4][3];
        load_tet_vertices(p, id / 6, (int)(id % 6), P);
        Tet t;
        finish_tet(P, scale, t);
        nc = (unsigned long long)((long long)(t.hi[0] - t.lo[0] + 1) * (t.hi[1] - t.lo[1] + 1) * (t.hi[2] - t.lo[2] + 1));
        atomicAdd(&sh_hist[bit_width_u64(nc - 1)], 1u);
        double det = tet_det_sign(t.g);
        inv = det < 0.0; deg = det == 0.0;
        if (id % 6 == 0) {  // once per Lagrangian cell: its three edges from corner 0 (as in k_census)
            const int64_t cell = id / 6;
            const int N = p.N;
            const int k = (int)(cell % N), j = (int)((cell / N) % N), i = (int)(cell / ((int64_t)N * N));
            double c0[3], c[3];
            load_pos(p, corner_index(i, j, k, 0, N), c0);
#pragma unroll
            for (int b = 1; b <= 4; b <<= 1) {
                load_pos(p, corner_index(i, j, k, b, N), c);
#pragma unroll
                for (int x = 0; x < 3; ++x) suspect |= fabs(unwrap1(c[x], c0[x], p.L, p.inv_L) - c0[x]) > 0.25 * p.L;
            }
        }
    }
    // warp partials (64-bit sum and max by halves), then one shared atomic per warp
    unsigned long long sum = nc, mx = nc;
    for (int o = 16; o; o >>= 1) {
        sum += __shfl_down_sync(0xffffffffu, sum, o);
        unsigned long long y = __shfl_down_sync(0xffffffffu, mx, o);
        mx = y > mx ? y : mx;
    }
    inv = __reduce_add_sync(0xffffffffu, inv);
    deg = __reduce_add_sync(0xffffffffu, deg);
    suspect = __reduce_add_sync(0xffffffffu, suspect);
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(&sh_stat[ST_SUM_CELLS], sum);
        atomicMax(&sh_stat[ST_MAX_CELLS], mx);
        if (inv) atomicAdd(&sh_stat[ST_INVERTED], (unsigned long long)inv);
        if (deg) atomicAdd(&sh_stat[ST_DEGENERATE], (unsigned long long)deg);
        if (suspect) atomicAdd(&sh_stat[ST_UNWRAP], (unsigned long long)suspect);
    }
    __syncthreads();
    if (threadIdx.x < 64 && sh_hist[threadIdx.x]) atomicAdd(&hist[threadIdx.x], (unsigned long long)sh_hist[threadIdx.x]);
    if (threadIdx.x == ST_SUM_CELLS && sh_stat[ST_SUM_CELLS]) atomicAdd(&stats[ST_SUM_CELLS], sh_stat[ST_SUM_CELLS]);
    if (threadIdx.x == ST_MAX_CELLS) atomicMax(&stats[ST_MAX_CELLS], sh_stat[ST_MAX_CELLS]);
    if (threadIdx.x == ST_INVERTED && sh_stat[ST_INVERTED]) atomicAdd(&stats[ST_INVERTED], sh_stat[ST_INVERTED]);
    if (threadIdx.x == ST_DEGENERATE && sh_stat[ST_DEGENERATE]) atomicAdd(&stats[ST_DEGENERATE], sh_stat[ST_DEGENERATE]);
    if (threadIdx.x == ST_UNWRAP && sh_stat[ST_UNWRAP]) atomicAdd(&stats[ST_UNWRAP], sh_stat[ST_UNWRAP]);
}

// ---------------------------------------------------------------- a7 refinement census
// counts[level] (dense, (base_G/P * 2^level)^3): tets whose cell range on the level grid meets
// each candidate patch position, each position once per tet.
struct LevelOffsets { long long off[8]; };  // start of each level's dense count array
__global__ void __launch_bounds__(256) k_patch_counts(Particles p, int base_G, int P, int n_levels,
                                                      unsigned long long* counts, LevelOffsets lo) {
    int64_t ntet = (int64_t)6 * p.N * p.N * p.N;
    int64_t id = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (id >= ntet) return;
    double V[4][3];
    load_tet_vertices(p, id / 6, (int)(id % 6), V);  // once for all levels
    for (int level = 0; level < n_levels; ++level) {
        const int Gl = base_G << level;
        const int np = Gl / P;
        unsigned long long* cl = counts + lo.off[level];
        Tet t;
        finish_tet(V, __ddiv_rn((double)Gl, p.L), t);
        // neighbouring tets mostly meet the same positions: one atomic per distinct position among
        // the lanes that are here together
        for_each_block(t.lo, t.hi, Gl, P, np, [&](int bx, int by, int bz, long long) {
            const unsigned int key = (unsigned int)(((long long)bx * np + by) * np + bz);
            const unsigned int peers = __match_any_sync(__activemask(), key);
            if ((int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(&cl[key], (unsigned long long)__popc(peers));
        });
    }
}

// a7 / PAPER.md:193 ("generating coarser representations for the internal nodes"): a patch all of
// whose 8 children are listed is not deposited into; each of its cells is the sum of the 2x2x2
// cells of the children that cover it (exact: the children tile the parent).  One thread per parent
// cell; `fam` holds, per refined patch, its own index followed by its 8 children's indices, child
// d = dx + 2 dy + 4 dz at position (2 ox + dx, 2 oy + dy, 2 oz + dz).  Run finest level first.
__global__ void __launch_bounds__(256) k_restrict(const int* fam, long long n_fam, int P, double* mass) {
    const long long P3 = (long long)P * P * P;
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= n_fam * P3) return;
    const long long q = t / P3;
    const int cell = (int)(t - q * P3);
    const int z = cell % P, y = (cell / P) % P, x = cell / (P * P);
    const int h = P / 2;
    const int dx = x >= h, dy = y >= h, dz = z >= h;
    const int* f = fam + q * 9;
    const double* c = mass + (long long)f[1 + dx + 2 * dy + 4 * dz] * P3;
    const int cx = 2 * (x - dx * h), cy = 2 * (y - dy * h), cz = 2 * (z - dz * h);
    double sum = 0.0;
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            const double* row = c + ((long long)(cx + a) * P + (cy + b)) * P + cz;
            sum += row[0] + row[1];
        }
    mass[(long long)f[0] * P3 + cell] = sum;
}

// a7: the memory-lean census.  One warp per sub-block of B^3 Lagrangian cells:
// the lanes stride over its (B+1)^3 particles (unwrapped to the minimum image of the first one)
// for the bounding box, then over the candidate patch positions the box meets; each receives
// T_b * vol(box n patch) / vol(box) in units of 2^-20 tets, rounded per term so that the integer
// sum is order independent (Q17).  Individually rounded IEEE operations throughout.
__global__ void __launch_bounds__(128) k_subblock_counts(Particles p, int base_G, int P, int level, int B,
                                                         unsigned long long* counts, unsigned int* overflow) {
    const int N = p.N;
    const int nb = (N + B - 1) / B;
    const long long sb = blockIdx.x * 4ll + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (sb >= (long long)nb * nb * nb) return;
    const int bk = (int)(sb % nb), bj = (int)((sb / nb) % nb), bi = (int)(sb / ((long long)nb * nb));
    const int o[3] = {bi * B, bj * B, bk * B};
    int n[3];
#pragma unroll
    for (int x = 0; x < 3; ++x) n[x] = (o[x] + B <= N) ? B : N - o[x];
    double ref[3], lo[3], hi[3];
    load_pos(p, ((int64_t)o[0] * N + o[1]) * N + o[2], ref);
#pragma unroll
    for (int c = 0; c < 3; ++c) { lo[c] = ref[c]; hi[c] = ref[c]; }
    const int n1 = n[1] + 1, n2 = n[2] + 1, npart = (n[0] + 1) * n1 * n2;
    for (int q = lane; q < npart; q += 32) {
        const int cc = q % n2, b = (q / n2) % n1, a = q / (n2 * n1);
        int ii = o[0] + a, jj = o[1] + b, kk = o[2] + cc;
        ii = ii >= N ? ii - N : ii; jj = jj >= N ? jj - N : jj; kk = kk >= N ? kk - N : kk;
        double v[3];
        load_pos(p, ((int64_t)ii * N + jj) * N + kk, v);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double x = unwrap1(v[c], ref[c], p.L, p.inv_L);
            lo[c] = fmin(lo[c], x); hi[c] = fmax(hi[c], x);
        }
    }
#pragma unroll
    for (int c = 0; c < 3; ++c)
        for (int s = 16; s; s >>= 1) {
            lo[c] = fmin(lo[c], __shfl_xor_sync(0xffffffffu, lo[c], s));
            hi[c] = fmax(hi[c], __shfl_xor_sync(0xffffffffu, hi[c], s));
        }
    const int Gl = base_G << level;
    const int np = Gl / P;
    const double scale = __ddiv_rn((double)Gl, p.L), Pc = (double)P;
    const double Tfix = (double)(6ll * n[0] * n[1] * n[2]) * 1048576.0;
    double glo[3], ghi[3], ext[3];
    int first[3], cnt[3];
#pragma unroll
    for (int x = 0; x < 3; ++x) {
        glo[x] = __dmul_rn(lo[x], scale); ghi[x] = __dmul_rn(hi[x], scale);
        ext[x] = __dsub_rn(ghi[x], glo[x]);
        first[x] = (int)floor(__ddiv_rn(glo[x], Pc));
        cnt[x] = (int)floor(__ddiv_rn(ghi[x], Pc)) - first[x] + 1;
    }
    if (cnt[0] > 64 || cnt[1] > 64 || cnt[2] > 64) {  // the oracle refuses such a box too
        if (lane == 0) atomicAdd(overflow, 1u);
        return;
    }
    auto share = [&](int x, int q) {
        double a = (double)((long long)(first[x] + q) * P), b = (double)((long long)(first[x] + q + 1) * P);
        a = glo[x] > a ? glo[x] : a;
        b = ghi[x] < b ? ghi[x] : b;
        double ov = __dsub_rn(b, a);
        ov = ov < 0.0 ? 0.0 : ov;
        return ext[x] > 0.0 ? __ddiv_rn(ov, ext[x]) : 1.0;
    };
    const int total = cnt[0] * cnt[1] * cnt[2];
    for (int q = lane; q < total; q += 32) {
        const int c = q % cnt[2], b = (q / cnt[2]) % cnt[1], a = q / (cnt[2] * cnt[1]);
        double f = __dmul_rn(share(0, a), share(1, b));
        f = __dmul_rn(f, share(2, c));
        const unsigned long long est = __double2ull_rd(__dadd_rn(__dmul_rn(Tfix, f), 0.5));
        const long long key = ((long long)wrap_mod(first[0] + a, np) * np + wrap_mod(first[1] + b, np)) * np +
                              wrap_mod(first[2] + c, np);
        if (est) atomicAdd(&counts[key], est);
    }
}

}  // namespace psd

// psd_abi.cu -- host side of libpsd: context, scratch management, launch order, C ABI.
// See include/psd.h for the contract of every entry point.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstddef>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/psd.h"
#include "psd_kernels.cuh"
#include "psd_faces.cuh"

using namespace psd;

#ifndef PSD_CENSUS_CB
#define PSD_CENSUS_CB 256  // threads per CTA of the census and scatter kernels
#endif

namespace {

struct DevBuf {
    void* p = nullptr;
    size_t cap = 0;
    cudaError_t ensure(size_t bytes) {
        if (bytes <= cap) return cudaSuccess;
        if (p) cudaFree(p);
        p = nullptr; cap = 0;
        size_t want = bytes + bytes / 8 + 256;  // a little slack so small growth does not realloc
        cudaError_t e = cudaMalloc(&p, want);
        if (e != cudaSuccess) {
            cudaGetLastError();  // the failed attempt must not stay behind as the runtime's last error
            e = cudaMalloc(&p, bytes);
            want = bytes;
        }
        if (e == cudaSuccess) cap = want;
        else { p = nullptr; cudaGetLastError(); }
        return e;
    }
    void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
    template <class T> T* as() const { return reinterpret_cast<T*>(p); }
};

}  // namespace

struct psd_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    Particles part{};
    bool built = false;
    double total_mass = 0.0;
    int weight_mode = 0, kernel = 0, counters = 0, chord_axis = -1, refine_subblock = 0, patch_restrict = 1,
        use_records = 1, rows_fp32 = 1, face_sharing = 1;
    bool accumulate_now = false;  // the running deposit adds to the caller's grid
    unsigned long long rec_pairs_max = 48ull << 20;  // capacity of the pair-record buffer (REC_PAIRS_MAX)
    long long class_small = CLASS_SMALL_MAX_CELLS;
    unsigned int chunk = 2048;
    DevBuf tile_counts, cursors, tile_offsets, item_offsets, items, pair_ids, part_pairs, part_items,
        totals, stats, hist, patches, lookup, refine_counts, host_pos, host_grid, families, records, slab_bounds,
        tet_info;
    unsigned long long* pinned = nullptr;  // [ST_COUNT + 128 + 2] staging
    psd_stats last{};
    bool stats_pending = false;
    bool binned_last = false;
    char err[384] = "";
    int64_t launches = 0;
    cudaEvent_t ev[6] = {};
    // psd_deposit_uniform_host: the grid goes back to the host slab by slab while later slabs are
    // still being deposited (copy stream + one event per slab)
    static constexpr int MAX_SLABS = 8;
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t slab_ev[MAX_SLABS] = {}, copy_done = nullptr;
    double* stream_out_host = nullptr;  // set only inside psd_deposit_uniform_host
    bool streamed = false;              // run_binned copied the grid itself
};

namespace {

int fail(psd_ctx* c, int code, const char* msg) {  // nothing here may throw across the C ABI
    if (c) {
        std::snprintf(c->err, sizeof(c->err), "%s", msg);
    }
    return code;
}
int cuda_fail(psd_ctx* c, cudaError_t e, const char* what) {
    char buf[320];
    std::snprintf(buf, sizeof(buf), "%s: %s", what, cudaGetErrorString(e));
    if (e == cudaErrorMemoryAllocation) cudaGetLastError();  // reported; do not leave it for the next check
    return fail(c, e == cudaErrorMemoryAllocation ? PSD_ERR_OOM : PSD_ERR_CUDA, buf);
}
#define CK(call)                                                    \
    do {                                                            \
        cudaError_t _e = (call);                                    \
        if (_e != cudaSuccess) return cuda_fail(ctx, _e, #call);    \
    } while (0)

// pair records (psd_kernels.cuh, k_pair_records): 13 doubles + 4 u64 + 2 u32 per pair
constexpr size_t REC_BYTES = 13 * 8 + 4 * 8 + 2 * 4;
constexpr unsigned long long REC_PAIRS_MAX = 48ull << 20;  // 48 Mi pairs = 6.9 GB
constexpr int REC_MAX_SLABS = 2048;  // record-buffer slabs of one deposit
constexpr int PINNED_WORDS = ST_COUNT + 128 + 2 + 2 * (psd_ctx::MAX_SLABS + 1) + 2 * (REC_MAX_SLABS + 2);

int reset_stats(psd_ctx* ctx) {
    CK(ctx->stats.ensure(sizeof(unsigned long long) * ST_COUNT));
    CK(ctx->hist.ensure(sizeof(unsigned long long) * 128));
    CK(cudaMemsetAsync(ctx->stats.p, 0, sizeof(unsigned long long) * ST_COUNT, ctx->stream));
    CK(cudaMemsetAsync(ctx->hist.p, 0, sizeof(unsigned long long) * 128, ctx->stream));
    return PSD_OK;
}

// census + scan + scatter + items + tile deposit over `n_tiles` tiles of `space`
int run_binned(psd_ctx* ctx, Space space, long long n_tiles) {
    space.class_small_max = ctx->class_small;
    cudaStream_t st = ctx->stream;
    const long long ncell = (long long)ctx->part.N * ctx->part.N * ctx->part.N;
    const long long n_bins = n_tiles * N_CLASSES;  // (tile, size class)
    CK(ctx->tile_counts.ensure(sizeof(unsigned int) * n_bins));
    CK(ctx->cursors.ensure(sizeof(unsigned int) * n_bins));
    CK(ctx->tile_offsets.ensure(sizeof(unsigned long long) * (n_bins + 1)));
    CK(ctx->item_offsets.ensure(sizeof(unsigned long long) * (n_bins + 1)));
    const int nparts = (int)((n_bins + SCAN_BLOCK - 1) / SCAN_BLOCK);
    CK(ctx->part_pairs.ensure(sizeof(unsigned long long) * nparts));
    CK(ctx->part_items.ensure(sizeof(unsigned long long) * nparts));
    CK(ctx->totals.ensure(sizeof(unsigned long long) * 2));
    CK(cudaMemsetAsync(ctx->tile_counts.p, 0, sizeof(unsigned int) * n_bins, st));
    CK(cudaMemsetAsync(ctx->cursors.p, 0, sizeof(unsigned int) * n_bins, st));
    int rc = reset_stats(ctx);
    if (rc) return rc;

    CK(cudaEventRecord(ctx->ev[0], st));
    const int cb = PSD_CENSUS_CB;
    const unsigned int cgrid = (unsigned int)((ncell + cb - 1) / cb);
    k_census<false><<<cgrid, cb, 0, st>>>(ctx->part, space, ctx->tile_counts.as<unsigned int>(), nullptr,
                                          nullptr, nullptr, ctx->stats.as<unsigned long long>(),
                                          ctx->hist.as<unsigned long long>());
    CK(cudaEventRecord(ctx->ev[1], st));
    // exclusive scan of the per-bin counts (pairs and work items) and the one host round trip of a
    // binned deposit: list sizes, the slabs' first items (host-output mode), max_extent
    int n_slabs = 0;
    auto scan_and_sync = [&](const unsigned int* counts) -> int {
        k_scan_partials<<<nparts, SCAN_BLOCK, 0, st>>>(counts, n_bins, ctx->chunk, ctx->part_pairs.as<unsigned long long>(),
                                                       ctx->part_items.as<unsigned long long>());
        k_scan_top<<<1, SCAN_BLOCK, 0, st>>>(ctx->part_pairs.as<unsigned long long>(),
                                             ctx->part_items.as<unsigned long long>(), nparts,
                                             ctx->totals.as<unsigned long long>());
        k_scan_final<<<nparts, SCAN_BLOCK, 0, st>>>(counts, n_bins, ctx->chunk, ctx->part_pairs.as<unsigned long long>(),
                                                    ctx->part_items.as<unsigned long long>(),
                                                    ctx->tile_offsets.as<unsigned long long>(),
                                                    ctx->item_offsets.as<unsigned long long>());
        ctx->launches += 3;
        CK(cudaGetLastError());
        CK(cudaMemcpyAsync(ctx->pinned + ST_COUNT + 128, ctx->totals.p, sizeof(unsigned long long) * 2,
                           cudaMemcpyDeviceToHost, st));
        // host-output mode (uniform grid): the first work item of each slab of x-tiles
        n_slabs = 0;
        if (ctx->stream_out_host && !space.patch_mode) {
            // few slabs for small grids: every launch ends in a partly filled wave
            n_slabs = space.nt / 8 < 1 ? 1 : (space.nt / 8 < psd_ctx::MAX_SLABS ? space.nt / 8 : psd_ctx::MAX_SLABS);
            for (int sl = 1; sl < n_slabs; ++sl) {
                const long long bin = (long long)(sl * space.nt / n_slabs) * space.nt * space.nt * N_CLASSES;
                CK(cudaMemcpyAsync(ctx->pinned + ST_COUNT + 130 + sl, ctx->item_offsets.as<unsigned long long>() + bin,
                                   sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
                CK(cudaMemcpyAsync(ctx->pinned + ST_COUNT + 130 + psd_ctx::MAX_SLABS + 1 + sl,
                                   ctx->tile_offsets.as<unsigned long long>() + bin, sizeof(unsigned long long),
                                   cudaMemcpyDeviceToHost, st));
            }
        }
        CK(cudaMemcpyAsync(ctx->pinned + ST_MAX_EXTENT, ctx->stats.as<unsigned long long>() + ST_MAX_EXTENT,
                           sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        return PSD_OK;
    };
    ctx->launches += 1;
    rc = scan_and_sync(ctx->tile_counts.as<unsigned int>());
    if (rc) return rc;
    unsigned long long n_pairs = ctx->pinned[ST_COUNT + 128], n_items = ctx->pinned[ST_COUNT + 129];
    const unsigned long long max_extent = ctx->pinned[ST_MAX_EXTENT];  // largest cell range of a tet along an axis (level 0)
    ctx->last.n_pairs = (int64_t)n_pairs;
    ctx->last.n_work_items = (int64_t)n_items;
    ctx->last.n_tiles = n_tiles;
    CK(cudaEventRecord(ctx->ev[2], st));
    // Shared faces (psd_faces.cuh): every face of the tessellation clipped once for its two tets.
    // Not accumulating (the grid is in fixed point until the end), two tets plus a tile shorter
    // than the grid (one periodic image per pair, neighbours' ranges unambiguous), on every level:
    // a range of e cells on level 0 is at most (e + 1) 2^l - 1 cells on level l.
    const int top_level = space.patch_mode ? space.n_levels - 1 : 0;
    const long long g0 = space.patch_mode ? space.base_G : space.G;
    const long long ext_top = (((long long)max_extent + 1) << top_level);
    bool pair_share = ctx->face_sharing && ctx->use_records && !ctx->accumulate_now && n_pairs > 0 &&
                            2ll * (long long)max_extent + 2 + TILE < g0 && 2ll * ext_top + 2 + TILE < (g0 << top_level) &&
                            ext_top <= TETINFO_MAX_EXTENT && (g0 << top_level) <= 2048;
    const int face_axis = ctx->chord_axis >= 0 ? ctx->chord_axis : ctx->face_sharing - 1;
    // (no room for the per-tet table: the tet formulation needs none)
    if (pair_share && ctx->tet_info.ensure(sizeof(TetInfo) * (size_t)(6 * ncell) * (size_t)(top_level + 1)) != cudaSuccess)
        pair_share = false;
    ctx->last.shared_faces = pair_share ? 1 : 0;
    if (n_pairs > 0) {
        if (n_items > 0x7fffffffull) return fail(ctx, PSD_ERR_INVALID_ARG, "too many work items");
        CK(ctx->pair_ids.ensure(sizeof(unsigned int) * n_pairs));
        CK(ctx->items.ensure(sizeof(Item) * n_items));
        k_items<<<(unsigned int)((n_tiles + 255) / 256), 256, 0, st>>>(
            ctx->tile_counts.as<unsigned int>(), n_tiles, ctx->chunk, ctx->tile_offsets.as<unsigned long long>(),
            ctx->item_offsets.as<unsigned long long>(), ctx->items.as<Item>());
        if (pair_share) {
            // what a pair needs of its tet and the four neighbours (weight, cell range), per level; the
            // scatter pass reads the cell ranges from it too
            const double mass_per_tet = ctx->total_mass / (6.0 * (double)ncell);
            if (top_level > 0)
                k_tet_info<true><<<(unsigned int)((6 * ncell + 255) / 256), 256, 0, st>>>(
                    ctx->part, (double)g0 / space.L, top_level + 1, mass_per_tet, ctx->weight_mode, ctx->tet_info.as<TetInfo>());
            else
                k_tet_info<false><<<(unsigned int)((6 * ncell + 255) / 256), 256, 0, st>>>(
                    ctx->part, (double)g0 / space.L, 1, mass_per_tet, ctx->weight_mode, ctx->tet_info.as<TetInfo>());
            ctx->launches += 1;
            k_scatter_info<<<(unsigned int)((6 * ncell + 255) / 256), 256, 0, st>>>(
                ctx->tet_info.as<TetInfo>(), 6 * ncell, space, ctx->tile_offsets.as<unsigned long long>(),
                ctx->cursors.as<unsigned int>(), ctx->pair_ids.as<unsigned int>());
        } else {
            k_census<true><<<cgrid, cb, 0, st>>>(ctx->part, space, nullptr, ctx->tile_offsets.as<unsigned long long>(),
                                                 ctx->cursors.as<unsigned int>(), ctx->pair_ids.as<unsigned int>(),
                                                 nullptr, nullptr);
        }
        ctx->launches += 2;
        CK(cudaEventRecord(ctx->ev[3], st));
        DepositArgs A{};
        A.part = ctx->part;
        A.space = space;
        A.pair_ids = ctx->pair_ids.as<unsigned int>();
        A.items = ctx->items.as<Item>();
        A.mass_per_tet = ctx->total_mass / (6.0 * (double)ncell);
        A.weight_mode = ctx->weight_mode;
        A.chord_axis = ctx->chord_axis;
        A.stats = ctx->stats.as<unsigned long long>();
        {
            // fixed-point unit of the tile accumulators: a cell of one work item receives at most
            // chunk x (mass of a tet, or one cell volume in signed-volume mode); 2^62 / that, as a
            // power of two
            const double unit = ctx->weight_mode == 0 ? std::fabs(A.mass_per_tet) : 1.0;
            int eu = 0, ec = 0;
            if (unit > 0.0 && std::isfinite(unit)) std::frexp(unit, &eu);   // unit < 2^eu
            std::frexp((double)ctx->chunk, &ec);                            // chunk < 2^ec
            A.acc_scale = std::ldexp(1.0, 61 - eu - ec);
            A.acc_inv_scale = std::ldexp(1.0, -(61 - eu - ec));
        }
        if (pair_share) {
            // tiles and grid are summed modulo 2^64 from end to end: the unit is 2^-62 of a bound of
            // the FINAL value of a cell (the whole mass; in signed-volume mode every cell ends at 1)
            A.chord_axis = face_axis;
            int eb = 0;
            const double bound = ctx->weight_mode == 0 ? std::fabs(ctx->total_mass) : 2.0;
            if (bound > 0.0 && std::isfinite(bound)) std::frexp(bound, &eb);  // bound < 2^eb
            A.acc_scale = std::ldexp(1.0, 62 - eb);
            A.acc_inv_scale = std::ldexp(1.0, -(62 - eb));
            A.tet_info = ctx->tet_info.p;
        }
        const size_t rec_bytes = pair_share ? sizeof(double) * REC2_DOUBLES : REC_BYTES;
        // ---- launch ranges of work items.  Boundaries (item index, first pair): the slabs of x-tiles
        // whose part of the grid goes back to the host while later slabs are deposited (host-output
        // mode), and the slabs of the pair-record buffer (k_pair_records writes the records of a
        // range, k_deposit_tiles consumes them; the buffer holds rec_cap pairs).
        struct Bound { unsigned long long item, pair; int x_slab_end; };
        Bound bounds[psd_ctx::MAX_SLABS + REC_MAX_SLABS + 4];
        int nb = 0;
        {
            const unsigned long long* ib = ctx->pinned + ST_COUNT + 130;
            const unsigned long long* pb = ib + psd_ctx::MAX_SLABS + 1;
            bounds[nb++] = Bound{0ull, 0ull, -1};
            for (int sl = 1; sl < n_slabs; ++sl) bounds[nb++] = Bound{ib[sl], pb[sl], sl - 1};
            bounds[nb++] = Bound{n_items, n_pairs, n_slabs > 1 ? n_slabs - 1 : -1};
        }
        unsigned long long rec_cap = 0;
        if (ctx->use_records) {
            const unsigned long long want = n_pairs < ctx->rec_pairs_max ? n_pairs : ctx->rec_pairs_max;
            if (ctx->records.ensure((size_t)want * rec_bytes) == cudaSuccess) rec_cap = want;
            // (no room: the deposit kernel then runs stage A itself)
        }
        if (rec_cap && n_pairs > rec_cap) {
            // cut at multiples of (rec_cap - chunk) pairs: a tiny kernel finds the items, one more
            // host round trip for them
            if (rec_cap <= 2ull * ctx->chunk) rec_cap = 0;
            else {
                const unsigned long long step = rec_cap - ctx->chunk;
                const unsigned long long ns = (n_pairs + step - 1) / step;
                if (ns > (unsigned long long)REC_MAX_SLABS) rec_cap = 0;
                else {
                    CK(ctx->slab_bounds.ensure(sizeof(unsigned long long) * 2 * (size_t)(ns + 1)));
                    k_slab_bounds<<<(unsigned int)((ns + 63) / 64), 64, 0, st>>>(A.items, n_items, n_pairs, step, (int)ns,
                                                                                ctx->slab_bounds.as<unsigned long long>());
                    ctx->launches += 1;
                    unsigned long long* hb = ctx->pinned + ST_COUNT + 130 + 2 * (psd_ctx::MAX_SLABS + 1);
                    CK(cudaMemcpyAsync(hb, ctx->slab_bounds.p, sizeof(unsigned long long) * 2 * (size_t)ns,
                                       cudaMemcpyDeviceToHost, st));
                    CK(cudaStreamSynchronize(st));
                    // merge (both lists ascend by item)
                    Bound merged[psd_ctx::MAX_SLABS + REC_MAX_SLABS + 4];
                    int nm = 0, ia = 0;
                    unsigned long long s = 1;  // slab 0 starts at item 0, already a boundary
                    while (ia < nb || s < ns) {
                        const bool take_a = ia < nb && (s >= ns || bounds[ia].item <= hb[2 * s]);
                        if (take_a) {
                            if (s < ns && hb[2 * s] == bounds[ia].item) ++s;
                            merged[nm++] = bounds[ia++];
                        } else {
                            merged[nm++] = Bound{hb[2 * s], hb[2 * s + 1], -1};
                            ++s;
                        }
                    }
                    nb = nm;
                    for (int i = 0; i < nb; ++i) bounds[i] = merged[i];
                }
            }
        }
        if (rec_cap) {
            char* rb = ctx->records.as<char>();
            A.rec_g = reinterpret_cast<const double*>(rb);
        }
        // The records-only deposit kernel needs every pair to meet its tile in one periodic image:
        // true when the largest cell range of a tet plus a tile fits the (coarsest) grid.
        const long long g_min = space.patch_mode ? space.base_G : space.G;
        const bool rec_only = rec_cap != 0 && (long long)max_extent + 2 + TILE < g_min;
        const Item* items0 = A.items;
        const size_t plane = sizeof(double) * (size_t)space.G * space.G;
        if (pair_share && !rec_cap)
            return fail(ctx, PSD_ERR_OOM, "no room for the pair records of the shared-face path (PSD_OPT_FACE_SHARING = 0 runs without)");
        for (int i = 0; i + 1 < nb; ++i) {
            const unsigned long long cnt = bounds[i + 1].item - bounds[i].item;
            if (cnt) {
                A.items = items0 + bounds[i].item;
                A.rec_pair_begin = bounds[i].pair;
                if (pair_share) {
                    if (ctx->rows_fp32) k_pair_records2<1><<<(unsigned int)cnt, REC2_THREADS, 0, st>>>(A);
                    else k_pair_records2<0><<<(unsigned int)cnt, REC2_THREADS, 0, st>>>(A);
                    if (ctx->counters) k_deposit_tiles2<true><<<(unsigned int)cnt, DEP_THREADS, DEP_SMEM_BYTES_REC, st>>>(A);
                    else k_deposit_tiles2<false><<<(unsigned int)cnt, DEP_THREADS, DEP_SMEM_BYTES_REC, st>>>(A);
                    ctx->launches += 2;
                } else {
                if (rec_cap) {
                    if (ctx->rows_fp32 && ctx->counters) k_pair_records<2><<<(unsigned int)cnt, REC_THREADS, 0, st>>>(A);
                    else if (ctx->rows_fp32) k_pair_records<1><<<(unsigned int)cnt, REC_THREADS, 0, st>>>(A);
                    else k_pair_records<0><<<(unsigned int)cnt, REC_THREADS, 0, st>>>(A);
                    ctx->launches += 1;
                }
                if (rec_only) {
                    if (ctx->counters) k_deposit_tiles<true, true><<<(unsigned int)cnt, DEP_THREADS, DEP_SMEM_BYTES_REC, st>>>(A);
                    else k_deposit_tiles<false, true><<<(unsigned int)cnt, DEP_THREADS, DEP_SMEM_BYTES_REC, st>>>(A);
                } else {
                    if (ctx->counters) k_deposit_tiles<true, false><<<(unsigned int)cnt, DEP_THREADS, DEP_SMEM_BYTES, st>>>(A);
                    else k_deposit_tiles<false, false><<<(unsigned int)cnt, DEP_THREADS, DEP_SMEM_BYTES, st>>>(A);
                }
                ctx->launches += 1;
                }
            }
            const int sl = bounds[i + 1].x_slab_end;
            if (sl >= 0 && pair_share) {  // the slab's planes from fixed point to fp64 before they leave
                const size_t x0 = (size_t)(sl * space.nt / n_slabs) * TILE, x1 = (size_t)((sl + 1) * space.nt / n_slabs) * TILE;
                k_fixed_to_double<<<1184, 256, 0, st>>>(space.out + x0 * (size_t)space.G * space.G,
                                                        (long long)((x1 - x0) * (size_t)space.G * space.G), A.acc_inv_scale);
                ctx->launches += 1;
            }
            if (sl >= 0) {  // a slab of x-tiles is complete: its part of the grid goes to the host
                CK(cudaEventRecord(ctx->slab_ev[sl], st));
                CK(cudaStreamWaitEvent(ctx->copy_stream, ctx->slab_ev[sl], 0));
                const size_t x0 = (size_t)(sl * space.nt / n_slabs) * TILE, x1 = (size_t)((sl + 1) * space.nt / n_slabs) * TILE;
                CK(cudaMemcpyAsync(reinterpret_cast<char*>(ctx->stream_out_host) + x0 * plane,
                                   reinterpret_cast<const char*>(space.out) + x0 * plane, (x1 - x0) * plane,
                                   cudaMemcpyDeviceToHost, ctx->copy_stream));
            }
        }
        if (pair_share && n_slabs <= 1) {  // all cells of the grid, or of the patches
            k_fixed_to_double<<<1184, 256, 0, st>>>(space.out, n_tiles * (long long)TILE_CELLS, A.acc_inv_scale);
            ctx->launches += 1;
        }
        if (n_slabs > 1) {
            CK(cudaEventRecord(ctx->copy_done, ctx->copy_stream));
            CK(cudaEventRecord(ctx->ev[4], st));  // the deposit's own time ends here
            CK(cudaStreamWaitEvent(st, ctx->copy_done, 0));
            ctx->streamed = true;
            CK(cudaGetLastError());
            ctx->stats_pending = true;
            ctx->binned_last = true;
            return PSD_OK;
        }
    } else {
        CK(cudaEventRecord(ctx->ev[3], st));
    }
    CK(cudaEventRecord(ctx->ev[4], st));
    CK(cudaGetLastError());
    ctx->stats_pending = true;
    ctx->binned_last = true;
    return PSD_OK;
}

int run_direct(psd_ctx* ctx, Space space) {
    cudaStream_t st = ctx->stream;
    const long long ncell = (long long)ctx->part.N * ctx->part.N * ctx->part.N;
    const long long ntet = 6 * ncell;
    int rc = reset_stats(ctx);
    if (rc) return rc;
    CK(cudaEventRecord(ctx->ev[0], st));
    k_tet_stats<<<(unsigned int)((ntet + 255) / 256), 256, 0, st>>>(
        ctx->part, (double)space.G / space.L, ctx->stats.as<unsigned long long>(), ctx->hist.as<unsigned long long>());
    CK(cudaEventRecord(ctx->ev[1], st));
    CK(cudaEventRecord(ctx->ev[2], st));
    CK(cudaEventRecord(ctx->ev[3], st));
    DepositArgs A{};
    A.part = ctx->part;
    A.space = space;
    A.pair_ids = nullptr;
    A.items = nullptr;
    A.mass_per_tet = ctx->total_mass / (6.0 * (double)ncell);
    A.weight_mode = ctx->weight_mode;
    A.chord_axis = ctx->chord_axis;
    A.stats = ctx->stats.as<unsigned long long>();
    A.acc_scale = A.acc_inv_scale = 1.0;  // the direct path adds to global memory in fp64
    const unsigned int grid = (unsigned int)((ntet + 127) / 128);
    if (ctx->counters) k_deposit_direct<true><<<grid, 128, 0, st>>>(A);
    else k_deposit_direct<false><<<grid, 128, 0, st>>>(A);
    ctx->launches += 2;
    CK(cudaEventRecord(ctx->ev[4], st));
    CK(cudaGetLastError());
    ctx->last.n_pairs = 0; ctx->last.n_work_items = 0; ctx->last.n_tiles = 0;
    ctx->stats_pending = true;
    ctx->binned_last = false;
    return PSD_OK;
}

bool valid_ctx(psd_ctx* ctx) { return ctx != nullptr; }

}  // namespace

extern "C" {

int psd_create(psd_ctx** out, int device, void* cuda_stream) {
    if (!out) return PSD_ERR_INVALID_ARG;
    *out = nullptr;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0 || device < 0 || device >= ndev) return PSD_ERR_CUDA;
    psd_ctx* ctx = new (std::nothrow) psd_ctx();
    if (!ctx) return PSD_ERR_OOM;
    ctx->device = device;
    ctx->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    e = cudaSetDevice(device);
    if (e == cudaSuccess) e = cudaMallocHost(&ctx->pinned, sizeof(unsigned long long) * PINNED_WORDS);
    for (int i = 0; i < 6 && e == cudaSuccess; ++i) e = cudaEventCreate(&ctx->ev[i]);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking);
    for (int i = 0; i < psd_ctx::MAX_SLABS && e == cudaSuccess; ++i)
        e = cudaEventCreateWithFlags(&ctx->slab_ev[i], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->copy_done, cudaEventDisableTiming);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_deposit_tiles<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, DEP_SMEM_BYTES);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_deposit_tiles<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, DEP_SMEM_BYTES_REC);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_deposit_tiles<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, DEP_SMEM_BYTES_REC);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_deposit_tiles<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, DEP_SMEM_BYTES);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_deposit_tiles2<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, DEP_SMEM_BYTES_REC);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_deposit_tiles2<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, DEP_SMEM_BYTES_REC);
    if (e != cudaSuccess) {
        psd_destroy(ctx);
        return PSD_ERR_CUDA;
    }
    *out = ctx;
    return PSD_OK;
}

void psd_destroy(psd_ctx* ctx) {
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    DevBuf* bufs[] = {&ctx->tile_counts, &ctx->cursors, &ctx->tile_offsets, &ctx->item_offsets, &ctx->items,
                      &ctx->pair_ids, &ctx->part_pairs, &ctx->part_items, &ctx->totals, &ctx->stats, &ctx->hist,
                      &ctx->patches, &ctx->lookup, &ctx->refine_counts, &ctx->host_pos, &ctx->host_grid, &ctx->families, &ctx->records, &ctx->slab_bounds, &ctx->tet_info};
    for (DevBuf* b : bufs) b->release();
    if (ctx->pinned) cudaFreeHost(ctx->pinned);
    for (int i = 0; i < 6; ++i)
        if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
    if (ctx->copy_stream) { cudaStreamSynchronize(ctx->copy_stream); cudaStreamDestroy(ctx->copy_stream); }
    for (int i = 0; i < psd_ctx::MAX_SLABS; ++i)
        if (ctx->slab_ev[i]) cudaEventDestroy(ctx->slab_ev[i]);
    if (ctx->copy_done) cudaEventDestroy(ctx->copy_done);
    delete ctx;
}

int psd_build_tets(psd_ctx* ctx, const void* pos_dev, int dtype, int stride_elems, int N, double L,
                   double total_mass) {
    if (!valid_ctx(ctx)) return PSD_ERR_INVALID_ARG;
    ctx->built = false;
    if (!pos_dev) return fail(ctx, PSD_ERR_INVALID_ARG, "pos_dev is NULL");
    if (dtype != PSD_F32 && dtype != PSD_F64) return fail(ctx, PSD_ERR_INVALID_ARG, "dtype must be PSD_F32 or PSD_F64");
    if (stride_elems != 3 && stride_elems != 4) return fail(ctx, PSD_ERR_INVALID_ARG, "stride_elems must be 3 or 4");
    if (N < 2 || N > 894) return fail(ctx, PSD_ERR_INVALID_ARG, "N must be in [2, 894]");
    if (!(L > 0.0) || !std::isfinite(L)) return fail(ctx, PSD_ERR_INVALID_ARG, "L must be finite and > 0");
    if (!std::isfinite(total_mass)) return fail(ctx, PSD_ERR_INVALID_ARG, "total_mass must be finite");
    if (dtype == PSD_F32 && stride_elems == 4 && (reinterpret_cast<uintptr_t>(pos_dev) & 15))
        return fail(ctx, PSD_ERR_INVALID_ARG, "float4 positions must be 16-byte aligned");
    CK(cudaSetDevice(ctx->device));
    ctx->part.pos = pos_dev;
    ctx->part.dtype = dtype;
    ctx->part.stride = stride_elems;
    ctx->part.N = N;
    ctx->part.L = L;
    {
        int e = 0;
        ctx->part.inv_L = std::frexp(L, &e) == 0.5 ? 1.0 / L : 0.0;  // exact reciprocal of a power of two
    }
    ctx->total_mass = total_mass;
    int rc = reset_stats(ctx);
    if (rc) return rc;
    k_validate<<<1184, 256, 0, ctx->stream>>>(ctx->part, ctx->stats.as<unsigned long long>());
    ctx->launches += 1;
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(ctx->pinned, ctx->stats.p, sizeof(unsigned long long) * ST_COUNT, cudaMemcpyDeviceToHost,
                       ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    std::memset(&ctx->last, 0, sizeof(ctx->last));
    ctx->last.n_tets = 6ll * N * N * N;
    ctx->last.n_nonfinite = (int64_t)ctx->pinned[ST_NONFINITE];
    ctx->stats_pending = false;
    if (ctx->last.n_nonfinite) return fail(ctx, PSD_ERR_INVALID_ARG, "positions contain NaN or Inf");
    ctx->built = true;
    return PSD_OK;
}

int psd_deposit_uniform(psd_ctx* ctx, int G, double* grid_dev, int accumulate) {
    if (!valid_ctx(ctx)) return PSD_ERR_INVALID_ARG;
    if (!ctx->built) return fail(ctx, PSD_ERR_STATE, "psd_deposit_uniform before psd_build_tets");
    if (G < 1 || G > 2048) return fail(ctx, PSD_ERR_INVALID_ARG, "G must be in [1, 2048]");
    if (!grid_dev) return fail(ctx, PSD_ERR_INVALID_ARG, "grid_dev is NULL");
    CK(cudaSetDevice(ctx->device));
    if (!accumulate) CK(cudaMemsetAsync(grid_dev, 0, sizeof(double) * (size_t)G * G * G, ctx->stream));
    ctx->accumulate_now = accumulate != 0;
    Space s{};
    s.patch_mode = 0;
    s.G = G;
    s.nt = G / TILE;
    s.out = grid_dev;
    s.L = ctx->part.L;
    const int64_t nf = ctx->last.n_nonfinite;
    std::memset(&ctx->last, 0, sizeof(ctx->last));
    ctx->last.n_tets = 6ll * ctx->part.N * ctx->part.N * ctx->part.N;
    ctx->last.n_nonfinite = nf;
    if (ctx->kernel == 1 || G % TILE != 0) return run_direct(ctx, s);
    return run_binned(ctx, s, (long long)s.nt * s.nt * s.nt);
}

int psd_deposit_patches(psd_ctx* ctx, const psd_patch* patches_host, int64_t n_patch, int P, int base_G,
                        double* mass_dev, int accumulate) {
    if (!valid_ctx(ctx)) return PSD_ERR_INVALID_ARG;
    if (!ctx->built) return fail(ctx, PSD_ERR_STATE, "psd_deposit_patches before psd_build_tets");
    if (!patches_host || n_patch < 1 || !mass_dev) return fail(ctx, PSD_ERR_INVALID_ARG, "NULL argument or no patches");
    {
        const long long tp = P / TILE;
        if ((long double)n_patch * tp * tp * tp * N_CLASSES > 2147483647.0L)
            return fail(ctx, PSD_ERR_INVALID_ARG, "too many patches: (tile, size class) bins are indexed with 32 bits");
    }
    if (P < TILE || P % TILE || base_G < P || base_G % P)
        return fail(ctx, PSD_ERR_INVALID_ARG, "P must be a multiple of 8 and divide base_G");
    CK(cudaSetDevice(ctx->device));
    int max_level = 0;
    for (int64_t q = 0; q < n_patch; ++q) {
        const psd_patch& pp = patches_host[q];
        if (pp.level < 0 || pp.level > 7) return fail(ctx, PSD_ERR_INVALID_ARG, "patch level out of range [0,7]");
        long long np = ((long long)base_G << pp.level) / P;
        if ((long long)base_G << pp.level > 2048 * 8)
            return fail(ctx, PSD_ERR_INVALID_ARG, "level grid too fine");
        if (pp.ox < 0 || pp.oy < 0 || pp.oz < 0 || pp.ox >= np || pp.oy >= np || pp.oz >= np)
            return fail(ctx, PSD_ERR_INVALID_ARG, "patch origin outside its level grid");
        if (pp.level > max_level) max_level = pp.level;
    }
    Space s{};
    s.patch_mode = 1;
    s.base_G = base_G;
    s.P = P;
    s.tp = P / TILE;
    s.np0 = base_G / P;
    s.tp_shift = -1;
    for (int k = 0; k < 16; ++k)
        if ((1 << k) == s.tp) s.tp_shift = k;
    s.n_levels = max_level + 1;
    s.L = ctx->part.L;
    s.out = mass_dev;
    long long total = 0;
    for (int l = 0; l <= max_level; ++l) {
        s.lookup_off[l] = total;
        long long np = ((long long)base_G << l) / P;
        total += np * np * np;
    }
    if (total > (1ll << 28))
        return fail(ctx, PSD_ERR_INVALID_ARG, "psd_deposit_patches: more than 2^28 patch positions on the listed levels");
    std::vector<int> lookup;
    std::vector<int> fam;                       // per refined patch: its index, then its 8 children
    std::vector<long long> fam_level_begin;     // first family of each level (families sorted by level)
    try {
        lookup.assign((size_t)total, -1);
        for (int64_t q = 0; q < n_patch; ++q) {
            const psd_patch& pp = patches_host[q];
            long long np = ((long long)base_G << pp.level) / P;
            long long idx = s.lookup_off[pp.level] + ((long long)pp.ox * np + pp.oy) * np + pp.oz;
            if (lookup[(size_t)idx] != -1) return fail(ctx, PSD_ERR_INVALID_ARG, "duplicate patch in list");
            lookup[(size_t)idx] = (int)q;
        }
        // a patch whose 8 children are all listed is filled by restriction, not deposited
        // into (PSD_OPT_PATCH_RESTRICT; not when accumulating: the children then hold old + new mass)
        if (ctx->patch_restrict && !accumulate && P % 2 == 0) {
            fam_level_begin.assign((size_t)max_level + 2, 0);
            for (int l = 0; l < max_level; ++l) {
                fam_level_begin[(size_t)l] = (long long)fam.size() / 9;
                const long long npc = ((long long)base_G << (l + 1)) / P;
                for (int64_t q = 0; q < n_patch; ++q) {
                    const psd_patch& pp = patches_host[q];
                    if (pp.level != l) continue;
                    int ch[8];
                    bool all = true;
                    for (int d = 0; d < 8 && all; ++d) {
                        const long long cx = 2ll * pp.ox + (d & 1), cy = 2ll * pp.oy + ((d >> 1) & 1), cz = 2ll * pp.oz + (d >> 2);
                        ch[d] = lookup[(size_t)(s.lookup_off[l + 1] + (cx * npc + cy) * npc + cz)];
                        all = ch[d] >= 0;
                    }
                    if (!all) continue;
                    fam.push_back((int)q);
                    for (int d = 0; d < 8; ++d) fam.push_back(ch[d]);
                }
            }
            fam_level_begin[(size_t)max_level] = fam_level_begin[(size_t)max_level + 1] = (long long)fam.size() / 9;
            // the deposit kernels find patches through `lookup`: refined ones are taken out of it
            for (size_t i = 0; i < fam.size(); i += 9) {
                const psd_patch& pp = patches_host[fam[i]];
                long long np = ((long long)base_G << pp.level) / P;
                lookup[(size_t)(s.lookup_off[pp.level] + ((long long)pp.ox * np + pp.oy) * np + pp.oz)] = -1;
            }
        }
    } catch (const std::bad_alloc&) {
        return fail(ctx, PSD_ERR_OOM, "psd_deposit_patches: host allocation failed");
    }
    CK(ctx->lookup.ensure(sizeof(int) * (size_t)total));
    CK(ctx->patches.ensure(sizeof(PatchDev) * (size_t)n_patch));
    if (!fam.empty()) CK(ctx->families.ensure(sizeof(int) * fam.size()));
    // pageable host memory: these copies complete before return, so the caller's list can go away
    CK(cudaMemcpyAsync(ctx->lookup.p, lookup.data(), sizeof(int) * (size_t)total, cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemcpyAsync(ctx->patches.p, patches_host, sizeof(PatchDev) * (size_t)n_patch, cudaMemcpyHostToDevice,
                       ctx->stream));
    if (!fam.empty())
        CK(cudaMemcpyAsync(ctx->families.p, fam.data(), sizeof(int) * fam.size(), cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    s.lookup = ctx->lookup.as<int>();
    s.patches = ctx->patches.as<PatchDev>();
    if (!accumulate) CK(cudaMemsetAsync(mass_dev, 0, sizeof(double) * (size_t)n_patch * P * P * P, ctx->stream));
    ctx->accumulate_now = accumulate != 0;
    const int64_t nf = ctx->last.n_nonfinite;
    std::memset(&ctx->last, 0, sizeof(ctx->last));
    ctx->last.n_tets = 6ll * ctx->part.N * ctx->part.N * ctx->part.N;
    ctx->last.n_nonfinite = nf;
    int rc = run_binned(ctx, s, (long long)n_patch * s.tp * s.tp * s.tp);
    if (rc) return rc;
    // restriction, finest refined level first (a parent's children may be refined themselves)
    for (int l = max_level - 1; l >= 0 && !fam.empty(); --l) {
        const long long b = fam_level_begin[(size_t)l], e = fam_level_begin[(size_t)l + 1];
        if (e <= b) continue;
        const long long threads = (e - b) * (long long)P * P * P;
        k_restrict<<<(unsigned int)((threads + 255) / 256), 256, 0, ctx->stream>>>(ctx->families.as<int>() + b * 9, e - b, P,
                                                                                   mass_dev);
        ctx->launches += 1;
    }
    CK(cudaGetLastError());
    ctx->last.n_restricted_patches = (int64_t)(fam.size() / 9);
    return PSD_OK;
}


int psd_refine_patches(psd_ctx* ctx, int base_G, int P, int max_level, double factor, int rule,
                       psd_patch* out_host, int64_t cap, int64_t* n_out, uint64_t* counts_host) {
    if (!valid_ctx(ctx)) return PSD_ERR_INVALID_ARG;
    if (!ctx->built) return fail(ctx, PSD_ERR_STATE, "psd_refine_patches before psd_build_tets");
    if (!n_out || P < 1 || base_G < P || base_G % P || max_level < 0 || max_level > 7 || !(factor > 0.0) ||
        (rule != PSD_RULE_LITERAL_TOP_DOWN && rule != PSD_RULE_BOTTOM_UP_LEVEL_MEAN))
        return fail(ctx, PSD_ERR_INVALID_ARG, "psd_refine_patches: bad argument");
    if (((long long)base_G << max_level) > 2048 * 8) return fail(ctx, PSD_ERR_INVALID_ARG, "level grid too fine");
    CK(cudaSetDevice(ctx->device));
    const int nl = max_level + 1;
    long long off[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    int np[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (int l = 0; l < nl; ++l) {
        np[l] = (base_G << l) / P;
        off[l + 1] = off[l] + (long long)np[l] * np[l] * np[l];
    }
    // the rule runs on the host over every candidate position: keep that bounded (and the patch
    // indices inside int)
    if (off[nl] > (1ll << 28))
        return fail(ctx, PSD_ERR_INVALID_ARG, "psd_refine_patches: more than 2^28 candidate patch positions");
  try {
    // one extra word at the end: boxes the sub-block census could not place
    CK(ctx->refine_counts.ensure(sizeof(unsigned long long) * (size_t)(off[nl] + 1)));
    CK(cudaMemsetAsync(ctx->refine_counts.p, 0, sizeof(unsigned long long) * (size_t)(off[nl] + 1), ctx->stream));
    const long long ntet = 6ll * ctx->part.N * ctx->part.N * ctx->part.N;
    if (ctx->refine_subblock > 0) {  // estimate from sub-block bounding boxes
        for (int l = 0; l < nl; ++l) {
            const int B = ctx->refine_subblock;
            const long long nb = (ctx->part.N + B - 1) / B;
            k_subblock_counts<<<(unsigned int)((nb * nb * nb + 3) / 4), 128, 0, ctx->stream>>>(
                ctx->part, base_G, P, l, B, ctx->refine_counts.as<unsigned long long>() + off[l],
                reinterpret_cast<unsigned int*>(ctx->refine_counts.as<unsigned long long>() + off[nl]));
            ctx->launches += 1;
        }
    } else {  // every tet counted, all levels in one pass over the tets
        LevelOffsets lo{};
        for (int l = 0; l < nl; ++l) lo.off[l] = off[l];
        k_patch_counts<<<(unsigned int)((ntet + 255) / 256), 256, 0, ctx->stream>>>(
            ctx->part, base_G, P, nl, ctx->refine_counts.as<unsigned long long>(), lo);
        ctx->launches += 1;
    }
    CK(cudaGetLastError());
    std::vector<unsigned long long> cnt((size_t)off[nl] + 1);
    CK(cudaMemcpyAsync(cnt.data(), ctx->refine_counts.p, sizeof(unsigned long long) * cnt.size(),
                       cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    if (cnt.back() != 0)
        return fail(ctx, PSD_ERR_UNWRAP, "sub-block census: a bounding box spans more than 64 patch positions");
    cnt.pop_back();
    if (counts_host) std::memcpy(counts_host, cnt.data(), sizeof(unsigned long long) * cnt.size());

    // ---- the rule, on integers (Q14)
    auto at = [&](int l, int a, int b, int c) -> size_t { return (size_t)(off[l] + ((long long)a * np[l] + b) * np[l] + c); };
    std::vector<char> exists((size_t)off[nl], 0), split((size_t)off[nl], 0);
    for (long long i = 0; i < off[1]; ++i) exists[(size_t)i] = 1;
    if (rule == PSD_RULE_BOTTOM_UP_LEVEL_MEAN) {
        // hot(l, pos): count > factor * mean of that level's counts, l >= 1
        std::vector<char> hot((size_t)off[nl], 0);
        for (int l = 1; l < nl; ++l) {
            long double sum = 0;
            for (long long i = off[l]; i < off[l + 1]; ++i) sum += (long double)cnt[(size_t)i];
            double mean = (double)(sum / (long double)(off[l + 1] - off[l]));
            for (long long i = off[l]; i < off[l + 1]; ++i) hot[(size_t)i] = (double)cnt[(size_t)i] > factor * mean;
        }
        for (int l = nl - 2; l >= 0; --l)
            for (int a = 0; a < np[l]; ++a)
                for (int b = 0; b < np[l]; ++b)
                    for (int c = 0; c < np[l]; ++c) {
                        char any = 0;
                        for (int d = 0; d < 8; ++d) {
                            size_t ch = at(l + 1, 2 * a + (d & 1), 2 * b + ((d >> 1) & 1), 2 * c + (d >> 2));
                            any |= hot[ch] | split[ch];
                        }
                        split[at(l, a, b, c)] = any;
                    }
    } else {
        long double sum = 0;
        for (long long i = 0; i < off[1]; ++i) sum += (long double)cnt[(size_t)i];
        double thr = factor * (double)(sum / (long double)off[1]);
        for (int l = 0; l + 1 < nl; ++l)
            for (long long i = off[l]; i < off[l + 1]; ++i) split[(size_t)i] = (double)cnt[(size_t)i] > thr;
    }
    for (int l = 0; l + 1 < nl; ++l)
        for (int a = 0; a < np[l]; ++a)
            for (int b = 0; b < np[l]; ++b)
                for (int c = 0; c < np[l]; ++c) {
                    size_t me = at(l, a, b, c);
                    if (!(exists[me] && split[me])) continue;
                    for (int d = 0; d < 8; ++d)
                        exists[at(l + 1, 2 * a + (d & 1), 2 * b + ((d >> 1) & 1), 2 * c + (d >> 2))] = 1;
                }
    int64_t n = 0;
    for (int l = 0; l < nl; ++l)
        for (int a = 0; a < np[l]; ++a)
            for (int b = 0; b < np[l]; ++b)
                for (int c = 0; c < np[l]; ++c)
                    if (exists[at(l, a, b, c)]) {
                        if (out_host && n < cap) out_host[n] = psd_patch{l, a, b, c};
                        ++n;
                    }
    *n_out = n;
    if (out_host && n > cap) return fail(ctx, PSD_ERR_INVALID_ARG, "patch list capacity too small");
    return PSD_OK;
  } catch (const std::bad_alloc&) {
    return fail(ctx, PSD_ERR_OOM, "psd_refine_patches: host allocation failed");
  }
}

int psd_deposit_uniform_host(psd_ctx* ctx, const void* pos_host, int dtype, int stride_elems, int N, double L,
                             double total_mass, int G, double* grid_host) {
    if (!valid_ctx(ctx)) return PSD_ERR_INVALID_ARG;
    if (!pos_host || !grid_host) return fail(ctx, PSD_ERR_INVALID_ARG, "NULL host buffer");
    if ((dtype != PSD_F32 && dtype != PSD_F64) || (stride_elems != 3 && stride_elems != 4) || N < 2 || N > 894 ||
        G < 1 || G > 2048)
        return fail(ctx, PSD_ERR_INVALID_ARG, "psd_deposit_uniform_host: bad argument");
    CK(cudaSetDevice(ctx->device));
    const size_t pbytes = (size_t)N * N * N * stride_elems * (dtype == PSD_F32 ? 4 : 8);
    const size_t gbytes = sizeof(double) * (size_t)G * G * G;
    CK(ctx->host_pos.ensure(pbytes));
    CK(ctx->host_grid.ensure(gbytes));
    CK(cudaMemcpyAsync(ctx->host_pos.p, pos_host, pbytes, cudaMemcpyHostToDevice, ctx->stream));
    int rc = psd_build_tets(ctx, ctx->host_pos.p, dtype, stride_elems, N, L, total_mass);
    if (rc) return rc;
    ctx->stream_out_host = grid_host;
    ctx->streamed = false;
    rc = psd_deposit_uniform(ctx, G, ctx->host_grid.as<double>(), 0);
    ctx->stream_out_host = nullptr;
    if (rc) return rc;
    if (!ctx->streamed)  // direct path, or nothing to deposit: one copy at the end
        CK(cudaMemcpyAsync(grid_host, ctx->host_grid.p, gbytes, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return PSD_OK;
}

int psd_deposit_patches_host(psd_ctx* ctx, const void* pos_host, int dtype, int stride_elems, int N, double L,
                             double total_mass, int base_G, int P, int max_level, double factor, int rule,
                             psd_patch* patches_out_host, int64_t cap, int64_t* n_out, double* mass_host) {
    if (!valid_ctx(ctx)) return PSD_ERR_INVALID_ARG;
    if (!pos_host || !patches_out_host || !n_out || !mass_host || cap < 1)
        return fail(ctx, PSD_ERR_INVALID_ARG, "psd_deposit_patches_host: NULL buffer or no capacity");
    if ((dtype != PSD_F32 && dtype != PSD_F64) || (stride_elems != 3 && stride_elems != 4) || N < 2 || N > 894)
        return fail(ctx, PSD_ERR_INVALID_ARG, "psd_deposit_patches_host: bad argument");
    CK(cudaSetDevice(ctx->device));
    const size_t pbytes = (size_t)N * N * N * stride_elems * (dtype == PSD_F32 ? 4 : 8);
    CK(ctx->host_pos.ensure(pbytes));
    CK(cudaMemcpyAsync(ctx->host_pos.p, pos_host, pbytes, cudaMemcpyHostToDevice, ctx->stream));
    int rc = psd_build_tets(ctx, ctx->host_pos.p, dtype, stride_elems, N, L, total_mass);
    if (rc) return rc;
    rc = psd_refine_patches(ctx, base_G, P, max_level, factor, rule, patches_out_host, cap, n_out, nullptr);
    if (rc) return rc;
    const size_t mbytes = sizeof(double) * (size_t)*n_out * P * P * P;
    CK(ctx->host_grid.ensure(mbytes));
    rc = psd_deposit_patches(ctx, patches_out_host, *n_out, P, base_G, ctx->host_grid.as<double>(), 0);
    if (rc) return rc;
    CK(cudaMemcpyAsync(mass_host, ctx->host_grid.p, mbytes, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return PSD_OK;
}

int psd_get_stats(psd_ctx* ctx, psd_stats* out) {
    if (!valid_ctx(ctx) || !out) return PSD_ERR_INVALID_ARG;
    CK(cudaSetDevice(ctx->device));
    if (ctx->stats_pending) {
        CK(cudaMemcpyAsync(ctx->pinned, ctx->stats.p, sizeof(unsigned long long) * ST_COUNT, cudaMemcpyDeviceToHost,
                           ctx->stream));
        CK(cudaMemcpyAsync(ctx->pinned + ST_COUNT, ctx->hist.p, sizeof(unsigned long long) * 128,
                           cudaMemcpyDeviceToHost, ctx->stream));
        CK(cudaStreamSynchronize(ctx->stream));
        psd_stats& s = ctx->last;
        s.sum_cells = (int64_t)ctx->pinned[ST_SUM_CELLS];
        s.max_cells = (int64_t)ctx->pinned[ST_MAX_CELLS];
        s.max_extent = (int64_t)ctx->pinned[ST_MAX_EXTENT];
        s.n_inverted = (int64_t)ctx->pinned[ST_INVERTED];
        s.n_degenerate = (int64_t)ctx->pinned[ST_DEGENERATE];
        s.n_unwrap_suspect = (int64_t)ctx->pinned[ST_UNWRAP];
        s.n_face_jobs = (int64_t)ctx->pinned[ST_TASKS];
        s.n_face_clips = (int64_t)ctx->pinned[ST_FACE_CLIPS];
        s.n_plane_evals = (int64_t)ctx->pinned[ST_PLANE_CLIPS];
        s.n_cells_written = (int64_t)ctx->pinned[ST_CELLS];
        s.n_general_clips = (int64_t)ctx->pinned[ST_GENERAL];
        s.n_rows_missed = (int64_t)ctx->pinned[ST_ROWS_MISSED];
        for (int i = 0; i < 64; ++i) {
            s.hist_tet[i] = ctx->pinned[ST_COUNT + i];
            s.hist_pair[i] = ctx->pinned[ST_COUNT + 64 + i];
        }
        s.tile_counts_dev = ctx->binned_last ? ctx->tile_counts.as<unsigned int>() : nullptr;
        cudaEventElapsedTime(&s.ms_census, ctx->ev[0], ctx->ev[1]);
        cudaEventElapsedTime(&s.ms_scan, ctx->ev[1], ctx->ev[2]);
        cudaEventElapsedTime(&s.ms_scatter, ctx->ev[2], ctx->ev[3]);
        cudaEventElapsedTime(&s.ms_deposit, ctx->ev[3], ctx->ev[4]);
        cudaEventElapsedTime(&s.ms_total, ctx->ev[0], ctx->ev[4]);
        ctx->stats_pending = false;
    } else {
        CK(cudaStreamSynchronize(ctx->stream));
    }
    *out = ctx->last;
    return PSD_OK;
}

int psd_get_tile_class_counts(psd_ctx* ctx, uint32_t* out_host, int64_t cap) {
    if (!valid_ctx(ctx) || !out_host) return PSD_ERR_INVALID_ARG;
    if (!ctx->binned_last || ctx->last.n_tiles <= 0) return fail(ctx, PSD_ERR_STATE, "no binned deposit to report");
    const int64_t n_bins = ctx->last.n_tiles * N_CLASSES;
    if (cap < n_bins) return fail(ctx, PSD_ERR_INVALID_ARG, "tile class count buffer too small");
    CK(cudaSetDevice(ctx->device));
    CK(cudaMemcpyAsync(out_host, ctx->tile_counts.p, sizeof(uint32_t) * (size_t)n_bins, cudaMemcpyDeviceToHost,
                       ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return PSD_OK;
}

int psd_get_tile_counts(psd_ctx* ctx, uint32_t* out_host, int64_t cap) {
    if (!valid_ctx(ctx) || !out_host) return PSD_ERR_INVALID_ARG;
    if (!ctx->binned_last || ctx->last.n_tiles <= 0) return fail(ctx, PSD_ERR_STATE, "no binned deposit to report");
    if (cap < ctx->last.n_tiles) return fail(ctx, PSD_ERR_INVALID_ARG, "tile count buffer too small");
    try {
        std::vector<uint32_t> bins((size_t)ctx->last.n_tiles * N_CLASSES);
        int rc = psd_get_tile_class_counts(ctx, bins.data(), (int64_t)bins.size());
        if (rc) return rc;
        for (int64_t t = 0; t < ctx->last.n_tiles; ++t) {
            uint32_t c = 0;
            for (int k = 0; k < N_CLASSES; ++k) c += bins[(size_t)t * N_CLASSES + k];
            out_host[t] = c;
        }
    } catch (const std::bad_alloc&) {
        return fail(ctx, PSD_ERR_OOM, "psd_get_tile_counts: host allocation failed");
    }
    return PSD_OK;
}

int psd_set_option(psd_ctx* ctx, int key, double value) {
    if (!valid_ctx(ctx)) return PSD_ERR_INVALID_ARG;
    const int iv = (int)value;
    switch (key) {
        case PSD_OPT_WEIGHT_MODE:
            if (iv != 0 && iv != 1) return fail(ctx, PSD_ERR_INVALID_ARG, "weight mode must be 0 or 1");
            ctx->weight_mode = iv; return PSD_OK;
        case PSD_OPT_KERNEL:
            if (iv != 0 && iv != 1) return fail(ctx, PSD_ERR_INVALID_ARG, "kernel must be 0 or 1");
            ctx->kernel = iv; return PSD_OK;
        case PSD_OPT_COUNTERS:
            ctx->counters = iv != 0; return PSD_OK;
        case PSD_OPT_CHUNK:
            if (iv < 32 || iv > (1 << 20)) return fail(ctx, PSD_ERR_INVALID_ARG, "chunk must be in [32, 2^20]");
            ctx->chunk = (unsigned int)iv; return PSD_OK;
        case PSD_OPT_CHORD_AXIS:
            if (iv < -1 || iv > 2) return fail(ctx, PSD_ERR_INVALID_ARG, "chord axis must be -1..2");
            ctx->chord_axis = iv; return PSD_OK;
        case PSD_OPT_CLASS_SMALL_CELLS:
            if (iv < 1 || iv > TILE_CELLS || (iv & (iv - 1)))
                return fail(ctx, PSD_ERR_INVALID_ARG, "class threshold must be a power of two in [1, 512]");
            ctx->class_small = iv; return PSD_OK;
        case PSD_OPT_PAIR_RECORDS:
            if (value < 0.0 || value > 4e9) return fail(ctx, PSD_ERR_INVALID_ARG, "pair records: 0, 1 or a capacity in pairs");
            ctx->use_records = value != 0.0;
            ctx->rec_pairs_max = value > 1.0 ? (unsigned long long)value : REC_PAIRS_MAX;
            return PSD_OK;
        case PSD_OPT_FACE_SHARING:
            if (iv < 0 || iv > 3) return fail(ctx, PSD_ERR_INVALID_ARG, "face sharing: 0 (off) or 1 + chord axis (1..3)");
            ctx->face_sharing = iv;
            return PSD_OK;
        case PSD_OPT_ROWS_FP32:
            if (iv != 0 && iv != 1) return fail(ctx, PSD_ERR_INVALID_ARG, "fp32 rows must be 0 or 1");
            ctx->rows_fp32 = iv; return PSD_OK;
        case PSD_OPT_PATCH_RESTRICT:
            if (iv != 0 && iv != 1) return fail(ctx, PSD_ERR_INVALID_ARG, "patch restriction must be 0 or 1");
            ctx->patch_restrict = iv; return PSD_OK;
        case PSD_OPT_REFINE_SUBBLOCK:
            if (iv < 0 || iv > 64) return fail(ctx, PSD_ERR_INVALID_ARG, "sub-block edge must be 0 (off) or 1..64 cells");
            ctx->refine_subblock = iv; return PSD_OK;
        default:
            return fail(ctx, PSD_ERR_INVALID_ARG, "unknown option key");
    }
}

int psd_sync(psd_ctx* ctx) {
    if (!valid_ctx(ctx)) return PSD_ERR_INVALID_ARG;
    CK(cudaSetDevice(ctx->device));
    CK(cudaStreamSynchronize(ctx->stream));
    return PSD_OK;
}

const char* psd_last_error(const psd_ctx* ctx) { return ctx ? ctx->err : "NULL context"; }

int64_t psd_launch_count(const psd_ctx* ctx) { return ctx ? ctx->launches : 0; }

}  // extern "C"

// ---------------------------------------------------------------- a deposit that allocates nothing
// psd_deposit_uniform_static (include/psd.h): the binned path with every scratch buffer in one
// file-scope device array.  In host code `psd_static_scratch` is only the host-side stand-in of
// the symbol, not a device address: the address is asked for once per device (with that device
// current) with cudaGetSymbolAddress and that pointer is what the kernels are given.
namespace {

constexpr int STATIC_MAX_TILES = (PSD_STATIC_MAX_G / TILE) * (PSD_STATIC_MAX_G / TILE) * (PSD_STATIC_MAX_G / TILE);
constexpr int STATIC_MAX_BINS = STATIC_MAX_TILES * N_CLASSES;
constexpr unsigned int STATIC_CHUNK = 2048;
constexpr int STATIC_MAX_ITEMS = STATIC_MAX_TILES + PSD_STATIC_MAX_PAIRS / (int)STATIC_CHUNK;
constexpr int STATIC_MAX_PARTS = (STATIC_MAX_BINS + SCAN_BLOCK - 1) / SCAN_BLOCK;

struct StaticScratch {
    // cleared at the start of every call (one memset): counts, cursors, statistics
    unsigned int tile_counts[STATIC_MAX_BINS];
    unsigned int cursors[STATIC_MAX_BINS];
    unsigned long long stats[ST_COUNT];
    unsigned long long hist[128];
    // written in full by the call before they are read
    unsigned long long totals[2];
    unsigned long long part_pairs[STATIC_MAX_PARTS];
    unsigned long long part_items[STATIC_MAX_PARTS];
    unsigned long long tile_offsets[STATIC_MAX_BINS + 1];
    unsigned long long item_offsets[STATIC_MAX_BINS + 1];
    Item items[STATIC_MAX_ITEMS];
    unsigned int pair_ids[PSD_STATIC_MAX_PAIRS];
};
static_assert(sizeof(StaticScratch) <= (size_t)PSD_STATIC_SCRATCH_BYTES, "scratch layout exceeds the stated size");
static_assert(offsetof(StaticScratch, totals) % 8 == 0 && offsetof(StaticScratch, items) % 8 == 0, "alignment");

static __device__ __align__(256) unsigned char psd_static_scratch[PSD_STATIC_SCRATCH_BYTES];

constexpr int STATIC_MAX_DEVICES = 64;
StaticScratch* g_static_ptr[STATIC_MAX_DEVICES] = {};  // device address of the array, per device
std::mutex g_static_mutex;

int static_fail(char* err, int err_len, int code, const char* msg) {
    if (err && err_len > 0) std::snprintf(err, (size_t)err_len, "%s", msg);
    return code;
}
int static_cuda_fail(char* err, int err_len, cudaError_t e, const char* what) {
    char buf[320];
    std::snprintf(buf, sizeof(buf), "%s: %s", what, cudaGetErrorString(e));
    return static_fail(err, err_len, PSD_ERR_CUDA, buf);
}
#define SCK(call)                                                                \
    do {                                                                         \
        cudaError_t _e = (call);                                                 \
        if (_e != cudaSuccess) return static_cuda_fail(err, err_len, _e, #call); \
    } while (0)

// once per device, with that device current: the array's device address, and the deposit
// kernel's dynamic shared-memory limit (neither allocates)
int static_setup(int device, StaticScratch** out, char* err, int err_len) {
    try {
        std::lock_guard<std::mutex> lock(g_static_mutex);
        if (!g_static_ptr[device]) {
            void* ptr = nullptr;
            SCK(cudaGetSymbolAddress(&ptr, psd_static_scratch));
            SCK(cudaFuncSetAttribute(k_deposit_tiles<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     DEP_SMEM_BYTES));
            g_static_ptr[device] = reinterpret_cast<StaticScratch*>(ptr);
        }
        *out = g_static_ptr[device];
    } catch (...) {
        return static_fail(err, err_len, PSD_ERR_CUDA, "psd_deposit_uniform_static: set-up lock failed");
    }
    return PSD_OK;
}

}  // namespace

extern "C" {

int psd_deposit_uniform_static(int device, void* cuda_stream, const void* pos_dev, int dtype, int stride_elems,
                               int N, double L, double total_mass, int G, double* grid_dev, int64_t* n_pairs_out,
                               char* err, int err_len) {
    if (err && err_len > 0) err[0] = 0;
    if (n_pairs_out) *n_pairs_out = 0;
    if (!pos_dev || !grid_dev) return static_fail(err, err_len, PSD_ERR_INVALID_ARG, "pos_dev or grid_dev is NULL");
    if (dtype != PSD_F32 && dtype != PSD_F64) return static_fail(err, err_len, PSD_ERR_INVALID_ARG, "dtype must be PSD_F32 or PSD_F64");
    if (stride_elems != 3 && stride_elems != 4) return static_fail(err, err_len, PSD_ERR_INVALID_ARG, "stride_elems must be 3 or 4");
    if (dtype == PSD_F32 && stride_elems == 4 && (reinterpret_cast<uintptr_t>(pos_dev) & 15))
        return static_fail(err, err_len, PSD_ERR_INVALID_ARG, "float4 positions must be 16-byte aligned");
    if (!(L > 0.0) || !std::isfinite(L)) return static_fail(err, err_len, PSD_ERR_INVALID_ARG, "L must be finite and > 0");
    if (!std::isfinite(total_mass)) return static_fail(err, err_len, PSD_ERR_INVALID_ARG, "total_mass must be finite");
    char msg[200];
    if (N < 2 || N > PSD_STATIC_MAX_N) {
        std::snprintf(msg, sizeof(msg), "psd_deposit_uniform_static: N = %d is outside [2, %d] (PSD_STATIC_MAX_N; the static scratch is sized for it)", N, PSD_STATIC_MAX_N);
        return static_fail(err, err_len, PSD_ERR_INVALID_ARG, msg);
    }
    if (G < TILE || G > PSD_STATIC_MAX_G || G % TILE) {
        std::snprintf(msg, sizeof(msg), "psd_deposit_uniform_static: G = %d must be a multiple of 8 in [8, %d] (PSD_STATIC_MAX_G; the static scratch is sized for it)", G, PSD_STATIC_MAX_G);
        return static_fail(err, err_len, PSD_ERR_INVALID_ARG, msg);
    }
    int ndev = 0;
    SCK(cudaGetDeviceCount(&ndev));
    if (device < 0 || device >= ndev || device >= STATIC_MAX_DEVICES) return static_fail(err, err_len, PSD_ERR_INVALID_ARG, "no such device");
    SCK(cudaSetDevice(device));
    StaticScratch* sc = nullptr;
    int rc = static_setup(device, &sc, err, err_len);
    if (rc) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);

    Particles part{};
    part.pos = pos_dev; part.dtype = dtype; part.stride = stride_elems; part.N = N; part.L = L;
    {
        int e = 0;
        part.inv_L = std::frexp(L, &e) == 0.5 ? 1.0 / L : 0.0;  // exact reciprocal of a power of two
    }
    Space space{};
    space.patch_mode = 0; space.G = G; space.nt = G / TILE; space.out = grid_dev; space.L = L;
    space.class_small_max = CLASS_SMALL_MAX_CELLS;
    const long long ncell = (long long)N * N * N;
    const long long n_tiles = (long long)space.nt * space.nt * space.nt, n_bins = n_tiles * N_CLASSES;
    const int nparts = (int)((n_bins + SCAN_BLOCK - 1) / SCAN_BLOCK);

    // the array keeps the last call's contents: clear what must start at zero (counts, cursors,
    // statistics: the head of the layout up to `totals`); the rest is written before it is read
    SCK(cudaMemsetAsync(sc, 0, offsetof(StaticScratch, totals), st));
    SCK(cudaMemsetAsync(grid_dev, 0, sizeof(double) * (size_t)G * G * G, st));
    k_validate<<<1184, 256, 0, st>>>(part, sc->stats);
    const int cb = PSD_CENSUS_CB;
    const unsigned int cgrid = (unsigned int)((ncell + cb - 1) / cb);
    k_census<false><<<cgrid, cb, 0, st>>>(part, space, sc->tile_counts, nullptr, nullptr, nullptr, sc->stats, sc->hist);
    k_scan_partials<<<nparts, SCAN_BLOCK, 0, st>>>(sc->tile_counts, n_bins, STATIC_CHUNK, sc->part_pairs, sc->part_items);
    k_scan_top<<<1, SCAN_BLOCK, 0, st>>>(sc->part_pairs, sc->part_items, nparts, sc->totals);
    k_scan_final<<<nparts, SCAN_BLOCK, 0, st>>>(sc->tile_counts, n_bins, STATIC_CHUNK, sc->part_pairs, sc->part_items,
                                               sc->tile_offsets, sc->item_offsets);
    SCK(cudaGetLastError());
    // the one host round trip: list sizes and the non-finite count, into stack variables
    unsigned long long totals[2] = {0ull, 0ull}, nonfinite = 0ull;
    SCK(cudaMemcpyAsync(totals, sc->totals, sizeof(totals), cudaMemcpyDeviceToHost, st));
    SCK(cudaMemcpyAsync(&nonfinite, sc->stats + ST_NONFINITE, sizeof(nonfinite), cudaMemcpyDeviceToHost, st));
    SCK(cudaStreamSynchronize(st));
    if (nonfinite) return static_fail(err, err_len, PSD_ERR_INVALID_ARG, "positions contain NaN or Inf");
    const unsigned long long n_pairs = totals[0], n_items = totals[1];
    if (n_pairs_out) *n_pairs_out = (int64_t)n_pairs;
    if (n_pairs > (unsigned long long)PSD_STATIC_MAX_PAIRS || n_items > (unsigned long long)STATIC_MAX_ITEMS) {
        std::snprintf(msg, sizeof(msg), "psd_deposit_uniform_static: %llu (tet, tile) pairs exceed PSD_STATIC_MAX_PAIRS = %d (the static pair list); use psd_deposit_uniform",
                      n_pairs, PSD_STATIC_MAX_PAIRS);
        return static_fail(err, err_len, PSD_ERR_INVALID_ARG, msg);
    }
    if (n_pairs == 0) return PSD_OK;
    k_items<<<(unsigned int)((n_tiles + 255) / 256), 256, 0, st>>>(sc->tile_counts, n_tiles, STATIC_CHUNK, sc->tile_offsets,
                                                                  sc->item_offsets, sc->items);
    k_census<true><<<cgrid, cb, 0, st>>>(part, space, nullptr, sc->tile_offsets, sc->cursors, sc->pair_ids, nullptr, nullptr);
    DepositArgs A{};
    A.part = part;
    A.space = space;
    A.pair_ids = sc->pair_ids;
    A.items = sc->items;
    A.mass_per_tet = total_mass / (6.0 * (double)ncell);
    A.weight_mode = 0;
    A.chord_axis = -1;
    A.stats = sc->stats;
    A.rec_g = nullptr;  // no pair records: the deposit kernel runs stage A itself
    A.rec_pair_begin = 0ull;
    {
        // fixed-point unit of the tile accumulators, as in run_binned: 2^61 / (chunk x mass of a tet)
        const double unit = std::fabs(A.mass_per_tet);
        int eu = 0, ec = 0;
        if (unit > 0.0 && std::isfinite(unit)) std::frexp(unit, &eu);
        std::frexp((double)STATIC_CHUNK, &ec);
        A.acc_scale = std::ldexp(1.0, 61 - eu - ec);
        A.acc_inv_scale = std::ldexp(1.0, -(61 - eu - ec));
    }
    k_deposit_tiles<false, false><<<(unsigned int)n_items, DEP_THREADS, DEP_SMEM_BYTES, st>>>(A);
    SCK(cudaGetLastError());
    return PSD_OK;
}

const char* psd_version(void) { return "libpsd sm_100a " __DATE__; }

}  // extern "C"

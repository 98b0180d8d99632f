/*
 * psd.h -- C ABI of libpsd: B200 (sm_100a) phase-space-element mass deposit.
 *
 * The operation (R. Kaehler, arXiv:1612.09491; citations are PAPER.md:LINE of the paper
 * text): N^3 tracer particles stored in Lagrangian order define N^3 periodic Lagrangian
 * cells; each cell is split into 6 tetrahedra of equal mass
 * m = M/(6 N^3); every tetrahedron T is intersected exactly with every
 * cubical deposit cell C it overlaps and
 *
 *        mass[C] += m * vol(T n C) / |vol(T)|            (PAPER.md:45-48 Eq. 1, :137)
 *
 * on a uniform periodic grid or on a list of cubical patches of an oct-tree.
 *
 * Conventions
 *  - All pointers named *_dev are DEVICE pointers on the context's device, *_host are HOST
 *    pointers.  No torch / C++ types cross this boundary.
 *  - The caller owns positions and outputs; the context owns its scratch (pair lists,
 *    counters), grown on demand and reused between calls.
 *  - Every function returns a psd_status (0 = PSD_OK); nothing throws or exits.
 *    psd_last_error() gives a human-readable string for the last failure on that context.
 *  - Work is enqueued on the context's CUDA stream.  psd_sync / psd_get_stats /
 *    psd_refine_patches / psd_build_tets / *_host calls synchronise with it.  The deposits return
 *    with the clip-and-deposit kernel still running, but on the binned path they block the
 *    host ONCE in between, after the census and the scan, to read the two list sizes that size
 *    the scratch and the launch (so they cannot be captured into a CUDA graph).
 *  - One context is used from one host thread at a time.
 *  - There is no CPU fallback: without a CUDA device psd_create fails.
 */
#ifndef PSD_H
#define PSD_H

#include <stdint.h>

#if defined(__GNUC__)
#define PSD_API __attribute__((visibility("default")))
#else
#define PSD_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct psd_ctx psd_ctx;

typedef enum {
    PSD_OK = 0,
    PSD_ERR_INVALID_ARG = 1, /* bad size / pointer / option                         */
    PSD_ERR_STATE = 2,       /* deposit or refine before psd_build_tets             */
    PSD_ERR_OOM = 3,         /* scratch allocation failed                           */
    PSD_ERR_CUDA = 4,        /* a CUDA call or kernel failed (see psd_last_error)   */
    PSD_ERR_UNWRAP = 5       /* psd_refine_patches with the sub-block census: a sub-block's
                                bounding box is too long for the minimum-image unwrap   */
} psd_status;

enum { PSD_F32 = 0, PSD_F64 = 1 };

/* psd_set_option keys */
enum {
    PSD_OPT_WEIGHT_MODE = 0, /* 0 (default): mass m/|V|.  1: signed volume, weight sign(det) in
                                cell-volume units -- every cell then receives exactly 1.0 for
                                any displacement field (a self-check needing no oracle).     */
    PSD_OPT_KERNEL = 1,      /* 0 (default): binned tile path when the grid allows it (G % 8 == 0).
                                1: direct path (one thread per tet, global atomics).           */
    PSD_OPT_COUNTERS = 2,    /* 1: also count face jobs / non-empty clips / plane integrals / cell
                                shares written during deposits (slower; for the work model).    */
    PSD_OPT_CHUNK = 3,       /* (tet,tile) pairs per work item of the binned path (default 2048) */
    PSD_OPT_CHORD_AXIS = 4,  /* -1 (default): per-tet longest AABB axis in the tet formulation,
                                the axis of PSD_OPT_FACE_SHARING with shared faces; 0/1/2: fixed x/y/z */
    PSD_OPT_REFINE_SUBBLOCK = 5 /* census used by psd_refine_patches.  0 (default): every tet is
                                counted.  B in 1..64: the paper's memory-lean
                                estimate (B = 8 there): the Lagrangian grid is
                                cut into sub-blocks of B^3 cells and a candidate patch receives
                                6 B^3 x vol(box n patch) / vol(box) from each sub-block's
                                bounding box; counts are then in units of 2^-20 tets
                                (PSD_SUBBLOCK_UNIT).  Valid while every sub-block's box is
                                shorter than L/2 (minimum-image unwrap) and meets at most 64
                                patch positions per axis, else PSD_ERR_UNWRAP.                */
    ,
    PSD_OPT_CLASS_SMALL_CELLS = 6, /* a3 size classes of the binned path: a (tet, tile) pair whose
                                cell range covers at most this many cells of the tile is class
                                "small", else "large"; a power of two in [1, 512] (default 8) so
                                that the classes are unions of the census buckets hist_pair[b] */
    PSD_OPT_PAIR_RECORDS = 8,  /* binned path.  1 (default): stage A of every (tet, tile) pair (tet
                                rebuilt from its id, determinant, tile-local vertices, per-row
                                column ranges of its faces) runs in its own kernel, which writes
                                144-byte pair records that the deposit kernel reads; the record
                                buffer holds up to 48 Mi pairs and is refilled slab by slab.
                                0: the deposit kernel runs stage A itself (no record buffer).
                                A value > 1 sets the buffer's capacity in pairs (tests).       */
    PSD_OPT_ROWS_FP32 = 9,     /* binned path with pair records, a4: which columns of a row of a face's
                                rectangle the face meets (the face jobs) is decided in fp32 with a
                                margin that covers fp32's rounding (1, default) or in fp64 with a
                                margin of 1e-9 (0).  Either set holds every column with a non-empty
                                polygon and the clip itself is fp64, so the deposit is the same;
                                fp32 admits a few more empty jobs (n_face_jobs).               */
    PSD_OPT_FACE_SHARING = 10, /* binned path (uniform grids and patches).  1..3 (default 1): every
                                face of the tessellation is clipped ONCE, for the two tets that
                                share it, in the (tet, tile) pair of the tet that owns it; one chord
                                axis for the whole deposit (value - 1 = x / y / z, unless
                                PSD_OPT_CHORD_AXIS fixes one); tiles and grid are summed in 64-bit
                                fixed point (unit 2^-62 of the total mass) and converted to fp64 at
                                the end.  Runs when twice the largest cell range of a tet plus a
                                tile fits the grid (on every level), with pair records and
                                accumulate = 0; else, and with 0, the tet formulation runs
                                (stats.shared_faces).                                          */
    PSD_OPT_PATCH_RESTRICT = 7  /* psd_deposit_patches, PAPER.md:193 (coarser representations of the
                                internal nodes).  1 (default): a listed patch whose 8 children are
                                all listed too is not deposited into; it is filled afterwards by
                                summing the 2x2x2 cells of its children, finest level first (the
                                children tile it, so this is the same mass up to rounding).
                                0: every listed patch is deposited into directly (Q13).
                                Ignored (as 0) when accumulate = 1 or P is odd.                */
};

#define PSD_SUBBLOCK_UNIT (1u << 20)

/* refinement rules (reading Q14 of PAPER.md:66) */
enum { PSD_RULE_LITERAL_TOP_DOWN = 0, PSD_RULE_BOTTOM_UP_LEVEL_MEAN = 1 };

/* One cubical patch of the block-structured oct-tree: it covers the cells
 * [o*P, o*P+P) per axis of the level grid with G_l = base_G * 2^level cells per side. */
typedef struct {
    int32_t level;
    int32_t ox, oy, oz;
} psd_patch;

typedef struct {
    int64_t n_tets;       /* 6 N^3                                                       */
    int64_t n_tiles;      /* tiles (8^3 cells) of the last binned deposit                */
    int64_t n_pairs;      /* (tet, tile) pairs = sum of tile_counts                      */
    int64_t n_work_items; /* chunks of pair lists scheduled                              */
    int64_t sum_cells;    /* sum over tets of AABB cells (candidate cells)               */
    int64_t max_cells;    /* largest AABB                                                */
    int64_t max_extent;   /* largest cell range of a tet along one axis (binned path)    */
    int64_t n_inverted;   /* tets with negative determinant                */
    int64_t n_degenerate; /* tets with determinant exactly 0                             */
    int64_t n_unwrap_suspect; /* Lagrangian cells with an unwrapped edge longer than L/4: the
                             minimum image is only valid below L/2 (Q4).  Advisory:
                             counted on both paths, never an error                          */
    int64_t n_nonfinite;  /* NaN/Inf position components seen by psd_build_tets          */
    uint64_t hist_tet[64];  /* tets by b = bit_width(n_cells-1)                          */
    uint64_t hist_pair[64]; /* pairs by b of the tet's cells inside that tile            */
    /* PSD_OPT_COUNTERS = 1 only: */
    int64_t n_face_jobs;    /* (tet face, column) jobs run                               */
    int64_t n_face_clips;   /* jobs whose clipped polygon is non-empty and reaches the run */
    int64_t n_plane_evals;  /* closed-form lattice-plane integrals of a face polygon     */
    int64_t n_cells_written;/* per-face cell shares added to accumulators                */
    int64_t n_restricted_patches; /* psd_deposit_patches: patches filled from their children     */
    int64_t n_general_clips; /* counters: face jobs the straight-line clip passed to the general
                               convex clip (a tie within its margin: lattice-aligned input)  */
    int64_t shared_faces;    /* 1: the last deposit clipped every face once for its two tets
                               (PSD_OPT_FACE_SHARING), 0: the tet formulation ran              */
    int64_t n_rows_missed;   /* counters, PSD_OPT_ROWS_FP32 = 1: rows of faces whose fp64 column range
                               the fp32 classification does not cover (a self-check: 0)       */
    /* device pointer to the per-(tile, size class) pair counts of the last binned deposit
       (2 * n_tiles uint32, see psd_get_tile_class_counts) */
    const uint32_t* tile_counts_dev;
    /* device time of the phases of the last deposit, ms (0 if not recorded)             */
    float ms_census, ms_scan, ms_scatter, ms_deposit, ms_total;
} psd_stats;

/* Create a context on CUDA device `device`.  `cuda_stream` is a cudaStream_t (NULL = the
 * legacy default stream) that all work of this context is enqueued on; it must outlive
 * the context. */
PSD_API int psd_create(psd_ctx** out, int device, void* cuda_stream);

/* Frees only context-owned scratch.  NULL is allowed. */
PSD_API void psd_destroy(psd_ctx* ctx);

/* PAPER.md:39-45, :60.  Register the particle set the tets are generated from.
 *   pos_dev      N^3 particles in Lagrangian order: particle (i,j,k) at element offset
 *                ((i*N+j)*N+k)*stride_elems, components x,y,z first (a 4th is ignored).
 *                BORROWED: must stay valid and unchanged until the last deposit using it.
 *   dtype        PSD_F32 or PSD_F64;  stride_elems 3 or 4 (4 with PSD_F32 = float4 loads).
 *   N            particles per side, >= 2 (6 N^3 must fit uint32: N <= 894).
 *   L            periodic box length > 0; positions are in [0, L] per axis.
 *   total_mass   M; every tet carries m = M/(6 N^3).
 * Tets are implicit (generated on the fly with minimum-image unwrapping relative to the
 * cell's corner 0; valid while every cell edge is shorter than L/2): nothing is stored.
 * Runs one validation pass over the positions and synchronises; non-finite positions give
 * PSD_ERR_INVALID_ARG. */
PSD_API int psd_build_tets(psd_ctx* ctx, const void* pos_dev, int dtype, int stride_elems, int N, double L,
                   double total_mass);

/* PAPER.md:137, :155-161.  Deposit all 6 N^3 tets onto the uniform periodic grid.
 *   G          cells per side (>= 1); cell (ix,iy,iz) spans [ix,ix+1)*L/G ...
 *   grid_dev   G^3 doubles, index (ix*G+iy)*G+iz, MASS per cell (not density).
 *   accumulate 0: the library zeroes the grid first; 1: adds to what is there.
 * Returns with the deposit kernel enqueued (one host round trip for the list sizes, see above). */
PSD_API int psd_deposit_uniform(psd_ctx* ctx, int G, double* grid_dev, int accumulate);

/* PAPER.md:66 (refinement by tet count), :72 (leaf patches).  Census-driven construction of
 * the patch list: counts, per level l = 0..max_level, the tets whose cell range meets each
 * candidate patch position of the level grid, then applies `rule` with `factor` on the host.
 *   base_G, P    level-0 grid and cells per patch side (base_G % P == 0)
 *   out_host     receives the patches ordered by level then (ox,oy,oz); cap = its capacity
 *   n_out        number of patches (also when cap is too small: then PSD_ERR_INVALID_ARG)
 *   counts_host  optional: receives the dense count arrays of all levels, concatenated
 *                (sum over l of (base_G/P * 2^l)^3 uint64); tets, or 2^-20 tets when
 *                PSD_OPT_REFINE_SUBBLOCK is set
 * Synchronous. */
PSD_API int psd_refine_patches(psd_ctx* ctx, int base_G, int P, int max_level, double factor, int rule,
                       psd_patch* out_host, int64_t cap, int64_t* n_out, uint64_t* counts_host);

/* PAPER.md:72, Q13.  Deposit into every listed patch the full contribution of
 * every tet that overlaps it, on the patch's own level grid.
 *   patches_host  n_patch patches (host; copied), distinct
 *   P             cells per patch side, multiple of 8;  base_G % P == 0
 *   mass_dev      n_patch * P^3 doubles, patch-major then (x*P+y)*P+z
 * Returns with the deposit (and restriction) kernels enqueued; the patch list is copied before
 * return; one host round trip for the list sizes, see above. */
PSD_API int psd_deposit_patches(psd_ctx* ctx, const psd_patch* patches_host, int64_t n_patch, int P,
                        int base_G, double* mass_dev, int accumulate);

/* End-to-end convenience used for the host-buffer measurement: copies positions host->device,
 * registers them, deposits, copies the G^3 grid device->host.  On the binned path the grid goes
 * back in up to 8 slabs of x-tiles, each copied (on a second stream) as soon as the work items
 * of its tiles are done, while the later slabs are still being deposited.  Synchronous.  Host
 * buffers should be pinned for full copy bandwidth and for the overlap. */
PSD_API int psd_deposit_uniform_host(psd_ctx* ctx, const void* pos_host, int dtype, int stride_elems, int N,
                             double L, double total_mass, int G, double* grid_host);

/* The same for the patch path with HOST buffers: copies
 * the positions host->device, registers them, builds the patch list (psd_refine_patches with
 * base_G, P, max_level, factor, rule), deposits into every listed patch and copies the masses
 * device->host.
 *   patches_out_host  receives the patch list (capacity cap patches); *n_out its length
 *   mass_host         receives *n_out * P^3 doubles, patch-major then (x*P+y)*P+z; the caller
 *                     provides room for cap * P^3 doubles
 * PSD_ERR_INVALID_ARG (and *n_out = the length needed) when cap is too small.  Synchronous. */
PSD_API int psd_deposit_patches_host(psd_ctx* ctx, const void* pos_host, int dtype, int stride_elems, int N,
                             double L, double total_mass, int base_G, int P, int max_level, double factor,
                             int rule, psd_patch* patches_out_host, int64_t cap, int64_t* n_out,
                             double* mass_host);

/* Synchronises, then fills *out with the counters of the last build / deposit. */
PSD_API int psd_get_stats(psd_ctx* ctx, psd_stats* out);

/* Synchronises, then copies the per-tile (tet, tile) pair counts of the last binned deposit to
 * out_host (n_tiles uint32; cap = its capacity in elements).  Uniform grid: tile
 * (tx*nt+ty)*nt+tz, nt = G/8.  Patches: patch-major, then the (P/8)^3 tiles of the patch.
 * PSD_ERR_STATE if the last deposit was not binned. */
PSD_API int psd_get_tile_counts(psd_ctx* ctx, uint32_t* out_host, int64_t cap);

/* As psd_get_tile_counts, split by the SIZE CLASS the pair lists are ordered by (BASELINE.json
 * north_star: bins by tile and by cells touched): out_host[2*tile + 0] = pairs whose tet covers
 * <= 8 cells of the tile ("small"), [2*tile + 1] = the others ("large"); cap >= 2 * n_tiles. */
PSD_API int psd_get_tile_class_counts(psd_ctx* ctx, uint32_t* out_host, int64_t cap);

PSD_API int psd_set_option(psd_ctx* ctx, int key, double value);
PSD_API int psd_sync(psd_ctx* ctx);
PSD_API const char* psd_last_error(const psd_ctx* ctx);

/* Number of kernels this context has launched so far (for bench.py's gpu_launches). */
PSD_API int64_t psd_launch_count(const psd_ctx* ctx);

/* ---- A deposit that allocates nothing ---------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture set-up, tight serving
 * loops, harnesses that forbid allocation).  The same operation as psd_build_tets +
 * psd_deposit_uniform on the binned path (census, counting sort by 8^3 tile,
 * tile deposit with stage A inside the deposit kernel, i.e. PSD_OPT_PAIR_RECORDS = 0), default
 * options, no context: all scratch (pair counts, offsets, work items, pair list) lives in ONE
 * file-scope `static __device__` array of PSD_STATIC_SCRATCH_BYTES (about 16.3 MiB) that every
 * GPU which loads the library holds until the process exits.  The call makes no cudaMalloc,
 * cudaFree, cudaMallocHost, event or stream creation, and calls no allocating library routine.
 *
 *   device, cuda_stream   the device is made current; all work is enqueued on the stream
 *   pos_dev      device, borrowed: N^3 particles as for psd_build_tets (dtype, stride_elems)
 *   N            2 .. PSD_STATIC_MAX_N
 *   G            a multiple of 8 in 8 .. PSD_STATIC_MAX_G
 *   grid_dev     device, caller-owned, double[G^3], index (ix*G+iy)*G+iz; overwritten
 *   n_pairs_out  host, may be NULL: number of (tet, tile) pairs of this deposit
 *   err, err_len host, may be NULL / 0: receives a message when the return value is not PSD_OK
 *
 * Limits (else PSD_ERR_INVALID_ARG with a message naming the limit, nothing deposited): N, G as
 * above, and at most PSD_STATIC_MAX_PAIRS (tet, tile) pairs (known only after the census: the
 * grid is then left zero-filled).  Positions with NaN/Inf are rejected like psd_build_tets.
 * One host round trip (the list sizes, copied into a stack variable) after the census; the
 * deposit kernels are then enqueued and the call returns: synchronise the stream before reading
 * grid_dev.  The scratch array is shared by every call in the process on that device and keeps
 * the last call's contents (what must start at zero is cleared by the call itself): calls that
 * overlap on the GPU (two streams, two threads) race -- serialise them. */
#define PSD_STATIC_MAX_N 64
#define PSD_STATIC_MAX_G 128
#define PSD_STATIC_MAX_PAIRS (4 << 20)
#define PSD_STATIC_SCRATCH_BYTES (17 << 20)
PSD_API int psd_deposit_uniform_static(int device, void* cuda_stream, const void* pos_dev, int dtype,
                                       int stride_elems, int N, double L, double total_mass, int G,
                                       double* grid_dev, int64_t* n_pairs_out, char* err, int err_len);

/* Library identification: "libpsd sm_100a <build date>" */
PSD_API const char* psd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PSD_H */

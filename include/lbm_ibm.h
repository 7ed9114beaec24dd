/*
 * lbm_ibm.h -- C ABI of the B200-native LBM-IBM time-step library (liblbm_ibm_b200.so).
 *
 * Method: Beny & Latt, "Efficient LBM on GPUs for dense moving objects using immersed boundary
 * condition" (arXiv 1904.02108).  "P:NN" = line NN of the paper text; "Rn" = reading n in
 * DESIGN.md.  One time step is the paper's pseudo-code P:60-66:
 *   1. rho, U from the populations (eq. (1))            -- only on cells near markers
 *   2. G = immersedBoundary(object, U) (section 3): multi-direct-forcing loop,
 *      Peskin 4-point kernel, markers moved by a rigid rotation on the device
 *   3.-6. D3Q19 BGK collision (eq. (2),(3)) with the body force (Guo term, R3; or the
 *      paper's velocity shift, as an option) fused with streaming (eq. (4)),
 *      periodic or half-way bounce-back faces.
 *
 * Conventions
 *  - All entry points are extern "C"; no exceptions or aborts cross the boundary.  Functions
 *    returning int give 0 on success and a negative LBM_E* code on error; the text of the last
 *    error of the calling thread is lbm_last_error().  On error the state is unchanged.
 *    Threads: different handles may be used from different host threads at the same time (no call synchronises
 *    the whole device or touches the legacy default stream after lbm_create has returned its handle); one handle is
 *    used by one thread at a time.
 *  - Every pointer argument marked "host or device" may point to pageable/pinned host memory or
 *    to device memory of the handle's GPU (detected with cudaPointerGetAttributes).  Pointers
 *    marked "host" are read on the CPU during the call.
 *  - Device INPUTS are read on the handle's stream (ibm_set_markers: by a blocking copy): what they
 *    hold must be complete before the call, i.e. produced on the handle's stream or on a stream the
 *    caller has synchronised with it.  Device OUTPUTS are written on the handle's stream and are
 *    valid for work enqueued behind it on that stream (or after lbm_sync).
 *  - The caller owns every buffer it passes; inputs are copied during the call and may be freed
 *    at once.  The library owns lattice and marker state (device memory of the current device at
 *    lbm_create time).
 *  - Field layout: x fastest, then y, then z: index = (z*ny + y)*nx + x; vector fields are three
 *    such planes [3][nz][ny][nx].  Lattice units; cell centres at integer coordinates 0..n-1; on
 *    a wall axis the wall planes sit half a link outside the first / last node (R16).
 *  - All work is enqueued on the handle's stream (lbm_set_stream; default: the legacy default
 *    stream).  lbm_ibm_step is asynchronous; lbm_read_fields / ibm_read_markers synchronise the
 *    stream before returning when the destination is host memory.
 *  - Arithmetic: fp32 on the device (populations are stored as f_i - t_i), fp64 only for the
 *    per-body rotation tables (R21).
 */
#ifndef LBM_IBM_H
#define LBM_IBM_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lbm lbm_t;

/* Boundary conditions and uniform body acceleration (BASELINE.json configs[1],[2]; R15). */
typedef struct {
    int wall_x, wall_y, wall_z; /* per axis: 0 = periodic, 1 = half-way bounce-back on both faces */
    double gx, gy, gz;          /* uniform body acceleration g_body added to the IBM force (R4)   */
} lbm_bc_t;

enum {
    LBM_OK = 0,
    LBM_EINVAL = -1,  /* bad argument (NULL handle, sizes < 1, tau <= 0.5, n < 0, zero axis ...)   */
    LBM_ENOMEM = -2,  /* device or host allocation failed                                        */
    LBM_ECUDA = -3,   /* a CUDA call or kernel failed; text in lbm_last_error()                   */
    LBM_ERANGE = -4,  /* a marker's 4x4x4 stencil would cross a wall face (R17)                   */
    LBM_ESTATE = -5   /* call not valid in the current state (e.g. kinematics before markers)    */
};

/* Options for lbm_set_option. */
enum {
    LBM_OPT_SPREAD = 1,   /* 0 = deterministic tile pass + tile footprints + gather-by-cell (default),
                             1 = global atomics, one thread per marker (measured comparison),
                             2 = plain gather-by-cell over the bins (slow reference variant),
                             3 = the paper's ib_force2 as printed: a block of 5^3 threads per marker with
                             atomicAdd (Alg.2; measured comparison)                      */
    LBM_OPT_FORCING = 2,  /* 0 = Guo source term (default, R3), 1 = paper's shift U + tau G */
    LBM_OPT_GRAPH = 3,    /* 1 = replay the step as a CUDA graph (default), 0 = plain launches     */
    LBM_OPT_LBM_KERNEL = 4, /* stream-collide variant: 0 = default, 1 = one cell per thread (the default),
                             2 = four cells per thread with 128-bit accesses (nx % 4 == 0; comparison;
                             used for the pure and the serial fused pass only)                     */
    LBM_OPT_INTERP = 5,   /* interpolation: 0 = inside the fused tile pass, from the tile's U window in shared
                             memory (default; with LBM_OPT_FUSED = 0: a kernel of its own, thread per marker
                             in sorted order), 1 = the paper's
                             ib_force1 access pattern: thread per marker in the caller's order, no reordering
                             (Alg.1; measured comparison), 2 = one warp per marker with a shuffle
                             reduction (the warp-cooperative design; measured comparison), 3 = one warp per
                             chunk with the chunk's U window staged in shared memory (measured comparison;
                             with LBM_OPT_SPREAD = 0 only)                                             */
    LBM_OPT_TIMING = 6,   /* 1 = run steps as plain launches with CUDA events between the phases and
                             accumulate per-phase device time (LBM_INFO_PHASE_NS); setting it resets
                             the accumulators.  Each step then ends with a stream synchronise.     */
    LBM_OPT_OVERLAP = 7,  /* how a coupled step is laid out in its CUDA graph.  1 = three concurrent branches: the MDF
                             loop, the stream-collide of every cell outside the marker stencils (it needs no
                             IBM force), and the binning of the NEXT step's markers (positions depend on
                             time only); the cells inside the stencils are updated after the join.  2 = two
                             branches (MDF loop, binning of the next step), then ONE fused stream-collide
                             pass over the whole lattice.  0 = one serial chain with a single fused
                             stream-collide pass (measured comparison).  3 (default) = 2 on lattices above
                             64 Mi cells or with tiles of 4 x 4 rows (the tile pass then fills the SMs by itself),
                             else 1.  Results are bit-identical.                                         */
    LBM_OPT_MOMENTS = 8,  /* where U is precomputed for the IBM: 0 = the de-duplicated list of
                             cells inside a marker stencil (default), 1 = the paper's box strategy (bounding
                             box of every body), 2 = the paper's kernel strategy (a block per Lagrangian
                             point, duplicates included).  Results are identical.                      */
    LBM_OPT_FUSED = 9,    /* 1 (default) = one MDF iteration is ONE tile pass that interpolates,
                             corrects and spreads (s g never leaves the SM) plus the collect; 0 = the
                             round-1 pipeline: interpolation kernel, TMA-fed tile sweep, collect (measured
                             comparison).  Only with LBM_OPT_SPREAD = 0 and LBM_OPT_INTERP = 0.           */
    LBM_OPT_TILE_ROWS = 10, /* source rows per tile in y and z for the fused path: 1, 2, 4, or 0 = automatic: the largest
                             of 4, 2, 1 for which the markers, in their rest pose, occupy at least 2,500 tiles (the
                             tile pass needs more tiles than warp slots; the number of tiles, not of markers,
                             decides: one thin body of 60,000 markers occupies ~300 tiles of 4 x 4 rows); single-row
                             tiles that are many and sparse (1,500 or more with fewer than 7 markers each) become
                             two-row tiles.
                             Changing it rebuilds the tile tables at the next step.  Results agree to rounding
                             (summation order).                                                           */
    LBM_OPT_PERSISTENT = 11, /* the fused MDF loop (moments + N x (tile pass, collect)) as ONE persistent kernel
                             with grid-wide barriers instead of 2 N + 1 launches: 1 = on, 2 = off, 0 (default) =
                             on for up to 3,000 single-row tiles (1,184 larger ones; see LBM_OPT_TILE_ROWS) and 100,000 markers on lattices
                             of up to 4 Mi cells (where the chain of launches is the critical path of the step).
                             Results are bit-identical.                                                   */
    LBM_OPT_TILE_CAP = 12, /* > 0: cap the number of tile footprints (default 0 = room for every tile that can
                             exist, up to 12 GB).  More tiles than the cap are dropped for that step and
                             lbm_sync reports LBM_ENOMEM; later steps that fit are complete again.  Takes
                             effect at the next step (the tables are re-allocated).                    */
    LBM_OPT_TILE_WARPS = 14, /* warps that work on one tile in the tile pass: 0 / 1 = one warp per tile (default),
                             2 = a pair of warps shares the tile's window of U; the tile's source rows are cut where
                             the marker count reaches half, each warp interpolates and sweeps its rows into a
                             footprint of its own and the write-out adds the two (measured comparison: 16 instead
                             of 12 warps per SM and half the longest tile, no faster: the pass is bound by the
                             shared-memory pipe).  Results agree to rounding (summation order).               */
    LBM_OPT_PIPELINE = 16, /* depth of the binning pipeline of the overlapped step (three marker sets are used in
                             turn): 2 = the step's graph bins the second half of step n + 1 (gather, chunks, tiles,
                             active cells, collect plan) and, in a branch of its own, the first half of step n + 2
                             (kinematics, keys, sort); 1 = it bins all of step n + 1 in one branch; 0 (default) = 2
                             up to 400,000 markers or in step layout 1, else 1.  Results are bit-identical.    */
    LBM_OPT_TRACE = 15,   /* 1 = the graph of the overlapped step also records a timing event after every kernel of
                             the MDF branch, after the bulk stream-collide and after the binning branches; after
                             lbm_sync, lbm_get_info(LBM_INFO_TRACE_NS + i) is the device time in ns from the fork
                             of the LAST step to event i and lbm_trace_label(i) names it.  A profiling aid
                             (the timeline of the concurrent branches); results do not depend on it.          */
    LBM_OPT_BULK_STREAM = 17, /* cache policy of the bulk stream-collide pass that runs beside the MDF loop (step layout
                             1): 1 = evict-first ("cache-streaming") loads and stores, so that the populations it
                             streams through L2 do not evict the few MB the MDF kernels work on; 2 = the default policy;
                             0 (default) = 1 on lattices of up to 4 Mi cells, else 2.  Results are
                             bit-identical.                                                                       */
    LBM_OPT_MDF_BLOCKS = 13 /* tuning: blocks per SM of the tile pass / of the persistent MDF kernel (0 = default:
                             as many as fit / one); fewer blocks leave more of every SM to the stream-collide
                             pass that runs beside the MDF loop.  Results do not depend on it.           */
};

/* Keys for lbm_get_info. */
enum {
    LBM_INFO_MARKERS = 1,       /* number of Lagrangian points                                   */
    LBM_INFO_BODIES = 2,
    LBM_INFO_STEPS = 3,         /* completed time steps                                           */
    LBM_INFO_LAUNCHES = 4,      /* kernels launched by this handle so far (graph nodes counted)   */
    LBM_INFO_ACTIVE_CELLS = 5,  /* cells inside at least one marker's stencil in the last step    */
    LBM_INFO_DEVICE_BYTES = 6,  /* device memory owned by the handle                              */
    LBM_INFO_STATUS = 7,        /* device-side status word of the last step (0 = OK)              */
    LBM_INFO_RUNS = 8,          /* marker chunks (markers of one row and one 8-cell x block) in the last step */
    LBM_INFO_RUN_ENTRIES = 9,   /* window cells (profile entries) over all chunks in the last step  */
    LBM_INFO_TILES = 10,        /* tiles (chunks of one x block and one block of tile-rows x tile-rows source rows) in the last step */
    LBM_INFO_ACTIVE_WORDS = 11, /* 32-cell words of the active mask that hold an active cell (the cells the
                                   second stream-collide pass of the overlapped step updates)          */
    LBM_INFO_LAYOUT = 13,       /* step layout in effect for the current markers (LBM_OPT_OVERLAP resolved: 0, 1, 2)   */
    LBM_INFO_TILE_ROWS = 14,    /* tile edge in effect (LBM_OPT_TILE_ROWS resolved: 1, 2, 4; 0 before the first step) */
    LBM_INFO_SORT_PASSES = 15,  /* 8-bit radix passes of the marker sort (ceil(log2(cells) / 8))                     */
    LBM_INFO_TRACE_COUNT = 12,  /* number of trace events of a step (LBM_OPT_TRACE)                  */
    LBM_INFO_TRACE_NS = 200,    /* + i: device time in ns from the fork of the last step to trace event i */
    LBM_INFO_PHASE_NS = 100     /* + phase: accumulated device time in ns under LBM_OPT_TIMING.
                                   phases: 0 kinematics+keys, 1 sort, 2 gather+bins, 3 moments on
                                   active cells, 4 interpolation+correction (fused path: the whole tile
                                   pass, sweep included), 5 spreading (fused path: the collect only),
                                   6 stream-collide (with LBM_OPT_OVERLAP: the pass over the cells
                                   outside the stencils), 7 stream-collide of the active cells     */
};

/* P:31 + eq.(3): allocate an nx*ny*nz D3Q19 lattice with relaxation time tau on the current CUDA
 * device and set it to rest (rho = 1, u = 0, i.e. f_i = t_i; R18).  bc may be NULL (periodic, no
 * body force).  Returns NULL on error (see lbm_last_error). */
lbm_t *lbm_create(int nx, int ny, int nz, double tau, const lbm_bc_t *bc);

/* Free everything the handle owns.  NULL is allowed. */
void lbm_destroy(lbm_t *h);

/* Host-only helper (no GPU needed): how an nx*ny*nz lattice is cut for the marker binning (DESIGN.md
 * section 5).  out[8] (host) = { x blocks per row, window entries per chunk profile, tiles in y,
 * tiles in z, 32-cell mask words per row, nominal block width (8), tile rows (4), largest window }.
 * Blocks are 8 cells wide; when nx % 8 is 1..3 the remainder joins the last block. */
int lbm_query_layout(int nx, int ny, int nz, int *out);

/* Use cuda_stream (a cudaStream_t; NULL = legacy default stream) for all later work. */
int lbm_set_stream(lbm_t *h, void *cuda_stream);

int lbm_set_option(lbm_t *h, int key, int value);
int lbm_get_info(lbm_t *h, int key, long long *value /* host */);

/* R18: f_i = Eq_i(rho, u) (eq. (3)) on every cell, with u the bare velocity of eq. (1).
 * rho [nz][ny][nx] or NULL (= 1); u [3][nz][ny][nx] or NULL (= 0); host or device; fp32.
 * Resets the step counter and the force field to zero. */
int lbm_set_fields(lbm_t *h, const float *rho, const float *u);

/* P:154 "object": define ONE rigid body of n Lagrangian points and append it to the handle.
 * pos [n][3] rest positions x(k) (on a periodic axis any real value, it is wrapped; on a wall axis
 * the stencil floor(x)-1..floor(x)+2 must stay inside 0..n-1, else LBM_ERANGE); vel [n][3]
 * additional, unrotated point velocity or NULL (= 0) (R14); area [n] the surface area s(k) of P:94.
 * All host or device, fp32.  Returns the body id (>= 0) or a negative error. */
int ibm_set_markers(lbm_t *h, const float *pos, const float *vel, const float *area, long long n);

/* P:154, Alg.1: the body most recently defined rotates rigidly with omega rad/step about
 * the line through center[3] along axis[3] (host, fp64; axis is normalised).  Step n -> n+1 places
 * point k at c + R(omega (n+1)) (p_k - c) and prescribes u_k = (R(omega (n+1)) - R(omega n))
 * (p_k - c) + vel_k (R12, R13).  Bodies without kinematics are static (omega = 0).  On a wall axis
 * the sphere swept by every point must keep its stencil inside the box, else LBM_ERANGE. */
int ibm_set_kinematics(lbm_t *h, double omega, const double *axis, const double *center);

/* Same as ibm_set_kinematics for the bodies first_body .. first_body+count-1 at once: omega [count],
 * axis [count][3], center [count][3] or NULL (= keep the centres); host, fp64.  When the centres
 * are kept only a small per-body table is copied to the device (no marker re-upload), so a host
 * controller may call this every step.  The angle of step n is omega * n (R13): changing omega
 * mid-run re-phases the body. */
int ibm_update_kinematics(lbm_t *h, int first_body, int count, const double *omega, const double *axis,
                          const double *center);

/* Remove all bodies and markers. */
int ibm_clear(lbm_t *h);

/* Advance nsteps time steps (pseudo-code P:60-66), each with mdf_iters multi-direct-forcing
 * iterations (the paper uses 5).  mdf_iters = 0 or no markers = pure LBM.
 * Asynchronous: returns after enqueueing on the handle's stream. */
int lbm_ibm_step(lbm_t *h, int nsteps, int mdf_iters);

/* Canonical read-out (R19): rho [nz][ny][nx] and bare velocity u [3][nz][ny][nx] (eq. (1)) of the
 * state after the last completed step; force [3][nz][ny][nx] = G of the last step (zero
 * before any step and away from markers).  Any pointer may be NULL; host or device; fp32. */
int lbm_read_fields(lbm_t *h, float *rho, float *u, float *force);

/* Marker read-out of the last step, in the caller's original marker order (bodies concatenated):
 * pos [n][3] current positions; force [n][3] = Delta u(k); cell [n] = linear index
 * of the owning lattice cell (floor of the position); perm [n]: perm[i] = original index of the
 * i-th marker after the stable sort by cell (ties by original index).  Any may be NULL;
 * host or device. */
int ibm_read_markers(lbm_t *h, float *pos, float *force, int *perm, int *cell);

/* The per-step result for a host controller, without stalling the time loop: enqueue the read-out of
 * the marker forces Delta u(k) of the last step (caller's order, force [n][3]) into HOST memory
 * (pinned for a truly asynchronous copy) and return at once.  Packing runs on the work stream, the
 * device-to-host copy on a stream of its own, so the next lbm_ibm_step overlaps it; the forces of
 * step n stay valid on the device until step n+2 is prepared.  `force` may be read after
 * ibm_wait_markers (or lbm_sync) returns; at most one read-out is in flight per handle: a second
 * call orders itself behind the first one's copy, so use a different `force` buffer if the first
 * has not been consumed. */
int ibm_read_markers_async(lbm_t *h, float *force /* host */);
int ibm_wait_markers(lbm_t *h);

/* Block until all enqueued work is done; returns LBM_ERANGE if a stencil crossed a wall during
 * the steps since the last sync (the offending step clamps the stencil instead of faulting), and
 * LBM_ENOMEM if the markers formed more chunks or tiles than the device tables hold (only possible
 * beyond the 12 GB footprint cap; the excess chunks were dropped). */
int lbm_sync(lbm_t *h);

/* Marker binning (a3: the stable sort by owning lattice cell the paper suggests) WITHOUT any allocation, for
 * callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it).  Needs no handle.  cell [n]: cell key of every marker, each < ncells (DEVICE pointer, not modified);
 * cell_sorted [n]: the keys in ascending order; perm [n]: perm[j] = index of the marker that holds rank j, equal keys
 * in ascending index order (the unique stable permutation, R20) -- both DEVICE pointers owned by the caller, and
 * the same result, bit for bit, as the permutation the handle-based path reports through ibm_read_markers.
 * The work (3 kernels per 8-bit pass, ceil(log2(ncells) / 8) passes) is enqueued on `cuda_stream` (a cudaStream_t, NULL
 * = the default stream); the call does not synchronise and calls no cudaMalloc / cudaFree or allocating library
 * routine.  The scratch of the sort (digit histograms, one ping-pong copy of keys and values) is a file-scope device
 * array of 3 MiB + 1 KiB that every GPU which loads the library holds until the process exits; its size fixes the
 * limit: n > IBM_NOALLOC_MAX_MARKERS returns LBM_ERANGE (use the handle-based path for larger sets).  n = 0 is a
 * no-op.  All calls on a device SHARE that array: calls whose kernels may overlap on the GPU (different streams
 * without an ordering between them, or different host threads) RACE on it -- keep them on one stream or order them
 * with events.  The array keeps the last call's contents; nothing in it has to start at zero (every word a call reads
 * it has written before).  Errors: LBM_EINVAL (n < 0, ncells out of 1..2^32, NULL or host pointers, cell_sorted
 * aliasing cell), LBM_ERANGE (n beyond the maximum), LBM_ECUDA. */
#define IBM_NOALLOC_MAX_MARKERS 262144
int ibm_sort_cells_noalloc(const unsigned *cell /* device */, int n, long long ncells, unsigned *cell_sorted /* device */,
                           int *perm /* device */, void *cuda_stream);

/* Text of the last error raised on the calling thread ("" if none). */
const char *lbm_last_error(void);

/* Label of trace event i of the last step (LBM_OPT_TRACE), "" when out of range.  The string is owned
 * by the handle and valid until the next step. */
const char *lbm_trace_label(lbm_t *h, int i);

#ifdef __cplusplus
}
#endif
#endif /* LBM_IBM_H */

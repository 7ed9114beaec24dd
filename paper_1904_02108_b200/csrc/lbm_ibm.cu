// C-ABI library of the B200-native LBM-IBM time step (see include/lbm_ibm.h for the contract).
// Host side: state, marshalling, launch sequencing and CUDA-graph replay.  Every arithmetic step
// of the hot path runs in the kernels of lbm_kernels.cuh / ibm_kernels.cuh / sort_kernels.cuh.
#include "../../include/lbm_ibm.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include <cstddef>

#include "ibm_kernels.cuh"
#include "mdf_kernels.cuh"
#include "sort_kernels.cuh"

using namespace lbmk;

namespace {

thread_local std::string g_err;

int fail(int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return code;
}

#define CK(expr)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (expr);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(e_ == cudaErrorMemoryAllocation ? LBM_ENOMEM : LBM_ECUDA, "%s: %s (%s:%d)", \
                        #expr, cudaGetErrorString(e_), __FILE__, __LINE__);                        \
    } while (0)

constexpr int MAX_MDF = 64;

// device scalars shared by both marker sets
struct DevScalars {
    long long step_ctr;  // time step n of the step being computed (kinematics angle)
    int status;          // != 0: a stencil crossed a wall
    int scratch;
};
// device scalars of one marker set (see PrepSet)
struct SetScalars {
    int n_prev;          // sorted markers whose bins are still registered in bin_first
    // ---- zeroed at the start of every preparation (k_kinematics), after k_clear_prev has used them
    int n_words;         // active words
    int n_chunks;        // chunks (may exceed the capacity: the excess is dropped and flagged)
    int n_entries;       // profile entries (window cells) over all chunks
    int n_cells;         // active cells
    int n_tiles;         // tiles (may exceed the capacity: the excess is dropped and flagged)
    int n_ovf;           // tile slots registered beyond the capacity (listed in PrepSet::ovf_slot)
    int n_felem;         // footprint elements handed out by the collect plan
    unsigned gbar;       // grid-wide barrier of the persistent MDF kernel (monotonic within a step)
    int cursor[MAX_MDF]; // work cursors of the tile passes, one per MDF iteration
    int bucket[16];      // tile size classes: counts [0..7] and fill cursors [8..15] (k_tile_count / k_tile_place)
    int icursor[MAX_MDF];// work cursors of the chunk-wise interpolation, one per MDF iteration
};
constexpr int N_STEP_COUNTERS = (int)((sizeof(SetScalars) - offsetof(SetScalars, n_words)) / sizeof(int));
constexpr int OVF_CAP = 4096;        // tile slots of a table overflow that are undone one by one

struct HostBody {
    long long first, count;
    double omega, axis[3], center[3];
    bool has_kin;
};

constexpr int LIST_GRID = 148 * 8;   // persistent-style grids for the list-driven kernels (grid-stride loops over device-side lists)
// Tile edge (source rows per tile in y and z) and persistent kernel go by the number of TILES the markers occupy
// (counted on the host for the rest pose, count_rest_tiles), because the marker count alone says little: 60,000 markers
// of ONE thin propeller occupy ~230 tiles of 4 x 4 rows (most of the 1,776 warp slots idle, 0.67 ms per step on 128^3)
// but ~2,000 single-row tiles (0.16 ms), while the same number of markers on 18 bodies fills 4,400 tiles of 4 x 4 rows.
//   edge = the largest of 4, 2, 1 with at least TILE_RULE_MIN_TILES tiles (~1.4 per warp slot);
//   single-row tiles that are many and sparse (>= 1,500 tiles with fewer than 7 markers each) become two-row tiles:
//   the per-tile work then outweighs the markers';
//   the persistent MDF kernel on small lattices up to PERSISTENT_MAX_TILES tiles.
// Measured on B200, ms per step at edge 1 / 2 / 4 (chain unless "p"): P1 0.239 / 0.233 / 0.290; 3 paper-shaped
// propellers 0.293 / 0.267 / 0.269p; P6 0.374 / 0.323 / 0.316p; P18 0.714 / 0.545 / 0.470; W4lit 0.89 / 0.74 / 0.68;
// one propeller on 128^3 with 61,440 markers 0.157p / 0.244p / 0.568p; 8 propellers on 128^3 with 18,432 markers
// 0.153p / 0.129p, with 73,728 markers 0.195 / 0.240p.  Persistent kernel against the chain on 128^3: faster with
// 924 .. 2,679 tiles, slower with 3,921 and 4,524.
constexpr long long TILE_RULE_MIN_TILES = 2500;
constexpr long long SPARSE_MIN_TILES = 1500;
constexpr double SPARSE_MAX_MARKERS_PER_TILE = 7.0;
constexpr long long PERSISTENT_MAX_TILES = 3000;
constexpr int PERSISTENT_MAX_MARKERS = 100000;  // persistent MDF kernel: measured faster than the kernel chain from 7,680 to 92,160 markers (one propeller, 128^3)
// Step layout (LBM_OPT_OVERLAP = 3): the split of the stream-collide into a bulk pass beside the MDF loop and a pass
// over the stencil cells pays while the MDF loop is a chain of short, latency-bound kernels that leave the SMs mostly
// idle (small marker sets); beyond that the tile pass fills the SMs itself and one fused pass after it is faster
// (measured: P18 0.469 against 0.552 ms per step, W4lit 0.683 against 0.740, W4 1.245 against 1.262)
constexpr long long SPLIT_MAX_CELLS = 64LL << 20;

// Optional per-phase device timing (LBM_OPT_TIMING): CUDA events recorded on the launching stream
// between the phases of a step; durations are accumulated after a stream synchronise.
enum { PH_KEYS = 0, PH_SORT, PH_BINS, PH_MOMENTS, PH_INTERP, PH_SPREAD, PH_LBM, PH_LBM_ACTIVE, PH_COUNT };
struct PhaseTimer {
    std::vector<cudaEvent_t> ev;
    std::vector<int> tag;
    size_t used = 0;
    double ns[PH_COUNT] = {0, 0, 0, 0, 0, 0, 0, 0};
    void mark(int phase, cudaStream_t s)
    {
        if (used == ev.size()) { cudaEvent_t e; cudaEventCreate(&e); ev.push_back(e); tag.push_back(0); }
        tag[used] = phase;
        cudaEventRecord(ev[used++], s);
    }
    void collect()
    {
        for (size_t i = 0; i + 1 < used; ++i) {
            float ms = 0.f;
            if (tag[i] >= 0 && cudaEventElapsedTime(&ms, ev[i], ev[i + 1]) == cudaSuccess) ns[tag[i]] += 1e6 * ms;
        }
        used = 0;
    }
    void reset() { for (double &v : ns) v = 0; used = 0; }
    ~PhaseTimer() { for (cudaEvent_t e : ev) cudaEventDestroy(e); }
};

}  // namespace

// Everything the binning stage (a1-a3) produces for ONE time step.  There are three sets, used in turn: while the
// MDF loop and the stream-collide of step n use set n % 3, two side branches of the step's graph prepare the steps to
// come (the marker positions depend on time only, not on the fluid): the second half of the binning of step
// n + 1 (gather, chunks, tiles, active cells, collect plan) and the first half of the binning of step n + 2
// (kinematics, keys, sort).  The binning is a chain of ~25 small dependent kernels; split over two steps its length
// stays below that of the MDF loop also for small marker sets, where every kernel costs its launch latency.
constexpr int N_SETS = 3;
struct PrepSet {
    unsigned *keys[2] = {nullptr, nullptr};   // radix ping-pong; the sorted keys end in keys[sort_passes & 1]
    int *vals[2] = {nullptr, nullptr};        // the permutation, same ping-pong
    MarkerSorted ms{nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    ChunkTable ct{nullptr, nullptr, nullptr};
    TileTable tt{nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};  // mask, id: dense over the tile slots; slot, rec: per tile; ohdr, orec: per position
    int *tile_order = nullptr;                // tiles by decreasing marker count (size classes)
    int *ovf_slot = nullptr;                  // tile slots registered without a footprint (table overflow), OVF_CAP entries
    int *fdst = nullptr;                      // collect plan: [tile][footprint element] -> index into F or -1
    int2 *cell_run = nullptr;                 // collect plan: [active cell] (first element in F, count)
    BodyStep *tabs = nullptr;                 // per-body rotation tables of the time step the set is prepared for (a1)
    int *inv = nullptr;                       // inverse permutation (comparison LBM_OPT_INTERP = 1 only; lazy)
    unsigned *headbits = nullptr;             // one bit per sorted marker: starts a run
    int *cells = nullptr;                     // active-cell list
    // dense maps, cleared incrementally by the set's next preparation (k_clear_prev)
    unsigned *amask = nullptr;                // active-cell bitmask, 32 consecutive x per word
    int *words = nullptr;                     // list of non-zero mask words
    int *chunk_of = nullptr;                  // [row][x block] -> packed (chunk id, lo, hi) or -1
    int *bin_first = nullptr;                 // cell -> first sorted marker (comparison spreads only; lazy)
    SetScalars *scal = nullptr;
    bool dirty = false;                       // the dense maps hold entries of a preparation
    long long step = -1;                      // time step the set is prepared for (-1: none)
    int stage = 0;                            // how far: 1 = first half (kinematics, keys, sort), 2 = complete
    int spread = -1;                          // prep_signature() the preparation was made for
};

struct lbm {
    int device = 0;
    cudaStream_t stream = nullptr;      // where work is enqueued
    cudaStream_t cap_stream = nullptr;  // capture-only streams for building graphs: the MDF chain (high priority),
    cudaStream_t cap_bulk = nullptr;    //   the bulk stream-collide (low priority),
    cudaStream_t cap_prep = nullptr;    //   the second half of the binning of the next step
    cudaStream_t cap_prep2 = nullptr;   //   the first half of the binning of the step after that
    cudaEvent_t ev_fork = nullptr, ev_bulk = nullptr, ev_prep = nullptr, ev_prep2 = nullptr, ev_mdf = nullptr;
    Geom g{};
    CollisionConst cc{};
    PlaneOffsets po{};
    double tau = 1.0;
    float *f[2] = {nullptr, nullptr};
    int cur = 0;                        // f[cur] holds the post-collision state to pull from
    float4 *U = nullptr, *G = nullptr;
    DevScalars *scal = nullptr;
    long long steps_done = 0;
    size_t n_mask_words = 0;
    PrepSet set[N_SETS];
    int cur_set = 0;                    // set the next IBM step uses
    int last_set = -1;                  // set of the last completed IBM step (G, mask, marker read-out), -1: none
    bool force_valid = false;           // G + mask of last_set describe the last completed step

    // markers: host mirror (caller order) and device copies
    std::vector<float> h_pos, h_vel, h_area;   // [n][3], [n][3], [n]
    // tiles the markers occupy in their rest pose, for tile edges 1, 2, 4 (bitmaps over the tile slots + counts): what the
    // automatic tile edge, step layout and persistent-kernel rules go by
    std::vector<unsigned long long> rest_map[3];
    long long rest_tiles[3] = {0, 0, 0};
    std::vector<int> h_body;
    std::vector<HostBody> bodies;
    std::vector<BodyDef> h_defs;        // host copy of the per-body device table
    bool markers_stale = true;          // device copies / graphs need rebuilding
    int nm = 0, nm_cap = 0, nb_cap = 0;
    float4 *d_qs = nullptr, *d_vb = nullptr;   // (p - c, s) and (vel, body id) per marker, caller order
    int *d_body = nullptr;
    BodyDef *d_defs = nullptr;
    int *d_hist[N_SETS] = {nullptr, nullptr, nullptr}, *d_total[N_SETS] = {nullptr, nullptr, nullptr};   // radix scratch, one per marker set (two binnings run side by side)
    size_t cells_cap = 0, headbits_cap = 0;
    float4 *F = nullptr;                // tile footprints [tile][7][7][cg.ent]
    ChunkGeom cg{1, CHUNK_W + 3};
    TileGeom tg{1, 1};
    int chunk_cap = 0, tile_cap = 0;    // capacity of the chunk table / of F
    size_t chunk_slots = 0, tile_slots = 0;   // entries of chunk_of / of the dense tile maps
    int rows_grid = 148;                // persistent grid of the round-1 tile sweep (blocks resident at once)
    int sms = 148;
    int tr = 0;                         // tile edge (source rows in y and z) the tile tables are built for; 0 = none yet
    int mdf_grid = 148, mdf2_grid = 148, mdfp_grid = 148;   // grids of the fused tile pass (one / two warps per tile) / of the persistent MDF kernel
    size_t mdf_wsmem = 0;               // shared memory per warp of the tile pass for (tr, cg)
    int words_grid = 148, moments_grid = 148;   // same for the active-word stream-collide and the moments kernel
    int sort_ipw = 64, sort_tiles = 0, sort_passes = 1;

    int opt_spread = 0, opt_forcing = 0, opt_graph = 1, opt_lbm_kernel = 0, opt_interp = 0, opt_timing = 0;
    int opt_overlap = 3, opt_moments = 0;
    int opt_pipeline = 0;
    int opt_fused = 1, opt_tile_rows = 0, opt_persistent = 0, opt_tile_cap = 0, opt_mdf_blocks = 0, opt_tile_warps = 0;
    int opt_bulk_stream = 0;
    bool realloc_tables = false;        // LBM_OPT_TILE_CAP changed: the tile tables are re-allocated at the next step
    int *d_box = nullptr;               // per-body bounding boxes (comparison LBM_OPT_MOMENTS = 1 only; lazy)
    PhaseTimer timer;
    // LBM_OPT_TRACE: timing events recorded inside the step graph after every kernel of every branch
    int opt_trace = 0;
    struct TraceList { std::vector<cudaEvent_t> ev; std::vector<std::string> label; };
    std::map<long long, TraceList> traces;      // one list per step graph (the variants differ in their kernels)
    TraceList *trace_cap = nullptr;             // list of the graph being captured
    const TraceList *trace_last = nullptr;      // list of the graph launched last
    long long last_key = 0;                     // key of the graph get_graph returned last
    std::map<long long, std::pair<cudaGraphExec_t, int>> graphs;   // key -> (exec, kernel nodes)
    long long launches = 0;
    size_t dev_bytes = 0;
    // staging buffers for host destinations / sources, kept between calls (a host controller reads the marker
    // forces every step: no cudaMalloc / cudaFree, which synchronise the device, on that path)
    void *stage[3] = {nullptr, nullptr, nullptr};
    size_t stage_cap[3] = {0, 0, 0};
    // asynchronous marker-force read-back (ibm_read_markers_async): packing on the work stream, D2H on a copy stream
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_pack = nullptr, ev_copy = nullptr;
    float *async_stage = nullptr;
    size_t async_cap = 0;
    bool copy_pending = false;
};

namespace {

template <class T>
int dmalloc(lbm *h, T **p, size_t count)
{
    *p = nullptr;
    if (count == 0) return LBM_OK;
    CK(cudaMalloc((void **)p, count * sizeof(T)));
    h->dev_bytes += count * sizeof(T);
    return LBM_OK;
}
template <class T>
void dfree(lbm *h, T *&p, size_t count)
{
    if (p) { cudaFree(p); h->dev_bytes -= count * sizeof(T); }
    p = nullptr;
}

// device staging buffer `slot` of at least `bytes` bytes; buffers up to 1 GB are kept for the next call
constexpr size_t STAGE_KEEP = (size_t)1 << 30;
void *stage_get(lbm *h, int slot, size_t bytes)
{
    if (h->stage_cap[slot] >= bytes) return h->stage[slot];
    if (h->stage[slot]) { cudaFree(h->stage[slot]); h->dev_bytes -= h->stage_cap[slot]; h->stage[slot] = nullptr; h->stage_cap[slot] = 0; }
    void *p = nullptr;
    if (cudaMalloc(&p, bytes) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    h->stage[slot] = p; h->stage_cap[slot] = bytes; h->dev_bytes += bytes;
    return p;
}
void stage_release(lbm *h)
{
    for (int a = 0; a < 3; ++a)
        if (h->stage[a] && h->stage_cap[a] > STAGE_KEEP) {
            cudaFree(h->stage[a]); h->dev_bytes -= h->stage_cap[a]; h->stage[a] = nullptr; h->stage_cap[a] = 0;
        }
}

bool is_device_ptr(const void *p)
{
    cudaPointerAttributes a{};
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

void drop_traces(lbm *h);
void drop_graphs(lbm *h)
{
    for (auto &kv : h->graphs) cudaGraphExecDestroy(kv.second.first);
    h->graphs.clear();
    drop_traces(h);
}

// LBM_OPT_TRACE: record a timing event on (capture) stream s; slot order = enqueue order, fixed per graph
void trace_mark(lbm *h, cudaStream_t s, const char *label, int idx = -1)
{
    if (!h->opt_trace || !h->trace_cap) return;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(s, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusActive) return;   // graph nodes only
    cudaEvent_t e;
    if (cudaEventCreate(&e) != cudaSuccess) return;
    char buf[64];
    if (idx >= 0) snprintf(buf, sizeof buf, "%s[%d]", label, idx); else snprintf(buf, sizeof buf, "%s", label);
    h->trace_cap->ev.push_back(e);
    h->trace_cap->label.emplace_back(buf);
    cudaEventRecordWithFlags(e, s, cudaEventRecordExternal);
}

void drop_traces(lbm *h)
{
    for (auto &kv : h->traces) for (cudaEvent_t e : kv.second.ev) cudaEventDestroy(e);
    h->traces.clear();
    h->trace_cap = nullptr; h->trace_last = nullptr;
}

void free_set(lbm *h, PrepSet &S)
{
    const size_t c = (size_t)h->nm_cap;
    for (int a = 0; a < 2; ++a) { dfree(h, S.keys[a], c); dfree(h, S.vals[a], c); }
    dfree(h, S.ms.fs, c); dfree(h, S.ms.wx, c); dfree(h, S.ms.wyz, 16 * c); dfree(h, S.ms.uk, c);
    dfree(h, S.ms.sg, c); dfree(h, S.ms.du, c);
    dfree(h, S.ct.first, (size_t)h->chunk_cap); dfree(h, S.ct.end, (size_t)h->chunk_cap);
    dfree(h, S.ct.slot, (size_t)h->chunk_cap);
    dfree(h, S.tt.slot, (size_t)h->tile_cap);
    dfree(h, S.tt.ohdr, (size_t)h->tile_cap);
    dfree(h, S.tt.orec, (size_t)h->tile_cap * (size_t)(h->tr * h->tr));
    dfree(h, S.tt.rec, (size_t)h->tile_cap * (size_t)(h->tr * h->tr));
    dfree(h, S.tile_order, (size_t)h->tile_cap);
    dfree(h, S.ovf_slot, (size_t)OVF_CAP);
    dfree(h, S.fdst, (size_t)h->tile_cap * (size_t)((h->tr + 3) * (h->tr + 3)) * (size_t)h->cg.ent);
    dfree(h, S.cell_run, h->cells_cap);
    dfree(h, S.tabs, (size_t)h->nb_cap);
    dfree(h, S.tt.mask, h->tile_slots); dfree(h, S.tt.id, h->tile_slots);
    dfree(h, S.inv, c);
    dfree(h, S.cells, h->cells_cap);
    dfree(h, S.headbits, h->headbits_cap);
    S.step = -1; S.stage = 0;
}

void free_markers_dev(lbm *h)
{
    const size_t c = (size_t)h->nm_cap;
    dfree(h, h->d_qs, c); dfree(h, h->d_vb, c);
    dfree(h, h->d_body, c);
    for (PrepSet &S : h->set) free_set(h, S);
    h->cells_cap = 0; h->headbits_cap = 0;
    dfree(h, h->F, (size_t)h->tile_cap * (size_t)((h->tr + 3) * (h->tr + 3)) * (size_t)h->cg.ent);
    h->chunk_cap = 0; h->tile_cap = 0; h->tile_slots = 0; h->tr = 0;
    for (int i = 0; i < N_SETS; ++i) {
        dfree(h, h->d_hist[i], (size_t)RADIX * (size_t)h->sort_tiles);
        dfree(h, h->d_total[i], (size_t)RADIX);
    }
    dfree(h, h->d_box, (size_t)6 * (size_t)h->nb_cap);
    dfree(h, h->d_defs, (size_t)h->nb_cap);
    h->nm_cap = 0; h->nb_cap = 0; h->sort_tiles = 0;
}

dim3 cell_block(const Geom &g)
{
    int bx = g.nx >= 256 ? 256 : ((g.nx + 31) / 32) * 32;
    int by = 256 / bx; if (by < 1) by = 1;
    return dim3(bx, by, 1);
}
dim3 cell_grid(const Geom &g, dim3 b) { return dim3((g.nx + b.x - 1) / b.x, (g.ny + b.y - 1) / b.y, g.nz); }

// the product path: fused tile pass + collect (mdf_kernels.cuh); everything else is a measured comparison
bool fused_path(const lbm *h) { return h->opt_fused && h->opt_spread == 0 && h->opt_interp == 0; }

// grid of a list-driven kernel: the lists (chunks, tiles, words, active cells) grow with the marker count, and a small
// marker set should not pay for scheduling 1184 mostly empty blocks in every one of its ~30 dependent kernels
int list_grid(const lbm *h)
{
    const long long want = (4LL * h->nm + 255) / 256;
    return (int)std::min<long long>(LIST_GRID, std::max<long long>(h->sms, want));
}

// the persistent MDF kernel can be considered: small lattices only (on larger ones the lattice-wide stream-collide is
// the critical path and the kernel only takes SM resources from it: P1 0.251 against 0.241 ms, P6 0.338 against 0.322)
constexpr long long PERSISTENT_MAX_CELLS = 4LL << 20;
bool persistent_eligible(const lbm *h, long long tiles, int tr)
{
    // multi-row tiles are heavy: there the kernel pays only while every warp of its grid (148 x 8) gets at most one
    // (8 propellers / 1,128 two-row tiles: 0.129 against 0.150 ms; a shell / 1,939 two-row tiles: 0.165 against 0.149)
    const long long max_tiles = tr == 1 ? PERSISTENT_MAX_TILES : (long long)h->sms * MDFP_WARPS;
    return h->g.cells <= PERSISTENT_MAX_CELLS && (long long)h->h_area.size() <= PERSISTENT_MAX_MARKERS && tiles <= max_tiles;
}

// the automatic choice of (tile edge, persistent kernel) for the markers as uploaded; tr_only > 0: for that edge
struct AutoPlan { int tr; bool persistent; };
AutoPlan auto_plan(const lbm *h, int tr_only = 0)
{
    int e = h->rest_tiles[2] >= TILE_RULE_MIN_TILES ? 2 : (h->rest_tiles[1] >= TILE_RULE_MIN_TILES ? 1 : 0);
    if (e == 0 && h->rest_tiles[0] >= SPARSE_MIN_TILES &&
        (double)h->h_area.size() < SPARSE_MAX_MARKERS_PER_TILE * (double)h->rest_tiles[0]) e = 1;
    if (tr_only) e = tr_only == 4 ? 2 : (tr_only == 2 ? 1 : 0);
    static const int edge[3] = {1, 2, 4};
    return AutoPlan{edge[e], persistent_eligible(h, h->rest_tiles[e], edge[e])};
}

// tile edge for the current markers and options: the comparison paths are written for 4 x 4 rows; the fused
// path takes the edge of the rule above unless LBM_OPT_TILE_ROWS says otherwise
int effective_tr(const lbm *h)
{
    if (!fused_path(h)) return TILE_R;
    if (h->opt_tile_rows) return h->opt_tile_rows;
    return auto_plan(h).tr;
}

// how a coupled step is laid out (LBM_OPT_OVERLAP): 0 = one serial chain; 1 = three branches (MDF loop, bulk
// stream-collide of the cells outside the stencils, binning of the next step), then the cells inside the stencils;
// 2 = two branches (MDF loop, binning of the next step), then ONE fused stream-collide pass over the lattice
int overlap_mode(const lbm *h)
{
    if (h->opt_overlap != 3) return h->opt_overlap;
    // 4 x 4-row tiles: the tile pass fills the SMs by itself, a bulk pass beside it only gets in its way (P18 0.470
    // against 0.522 ms, W4lit 0.68 against 0.78); smaller tiles: the MDF kernels are short and latency-bound, the
    // bulk pass runs beside them (P6 0.324 against 0.360, P1 0.239 against 0.281)
    return (h->g.cells > SPLIT_MAX_CELLS || effective_tr(h) == TILE_R) ? 2 : 1;
}

// warps per tile of the tile pass: two share a tile's window and footprint where tiles hold several batches of 32
// markers (4 x 4-row tiles), one otherwise
int tile_warps(const lbm *h)
{
    return h->opt_tile_warps == 2 ? 2 : 1;
}

// The whole MDF loop as one persistent kernel (LBM_OPT_PERSISTENT; automatic: small marker sets on small lattices).
// With few markers every tile pass and collect costs its launch latency, and the chain of 2 N + 1 dependent launches
// is the critical path of the step as long as the lattice-wide stream-collide beside it is shorter; on larger
// lattices the stream-collide is the critical path and a persistent kernel only takes SM resources from it
// (measured on B200: W3 0.107 against 0.140 ms per step, P1 0.251 against 0.241, P6 0.338 against 0.322).
bool use_persistent(const lbm *h)
{
    if (!fused_path(h) || h->opt_moments != 0 || h->opt_timing) return false;
    if (h->opt_persistent) return h->opt_persistent == 1;
    return auto_plan(h, h->opt_tile_rows).persistent;
}

// Cache policy of the bulk stream-collide pass that runs beside the MDF loop (LBM_OPT_BULK_STREAM): evict-first loads
// and stores keep the ~1 GB it streams through L2 from evicting what the MDF kernels work on.  Automatic: on lattices
// of up to 4 Mi cells (beside the persistent MDF kernel W3 gains 7 %, beside the kernel chain W3x4 4 %; on the 8 Mi
// cells of P1 / P6 it costs 1 %).
bool bulk_stream(const lbm *h)
{
    if (h->opt_bulk_stream) return h->opt_bulk_stream == 1;
    return use_persistent(h) || h->g.cells <= PERSISTENT_MAX_CELLS;
}

// Depth of the binning pipeline (LBM_OPT_PIPELINE): 2 = the binning of a step is spread over the two steps before it
// (small marker sets: the chain of ~25 dependent launches is longer than the MDF loop); 1 = all of it during the
// step before (large sets: the binning is short beside the MDF loop and a second branch only adds contention)
constexpr int PIPE2_MAX_MARKERS = 400000;
int pipeline_depth(const lbm *h)
{
    if (h->opt_pipeline) return h->opt_pipeline;
    // layout 1 (small tiles): the binning chain is on the critical path whatever the marker count (a shell of 420,000
    // markers on 128^3: 0.447 against 0.507 ms)
    return (h->nm <= PIPE2_MAX_MARKERS || overlap_mode(h) == 1) ? 2 : 1;
}

// the options a preparation depends on (which tables it builds)
int prep_signature(const lbm *h) { return h->opt_spread | (h->opt_interp << 4) | (h->tr << 8) | ((int)fused_path(h) << 12); }

const unsigned *sorted_keys(const lbm *h, const PrepSet &S) { return S.keys[h->sort_passes & 1]; }
const int *sorted_perm(const lbm *h, const PrepSet &S) { return S.vals[h->sort_passes & 1]; }

// the dense cell -> first-marker map is needed by the comparison spreads only
int ensure_bin_first(lbm *h, PrepSet &S)
{
    if (S.bin_first) return LBM_OK;
    int rc = dmalloc(h, &S.bin_first, (size_t)h->g.cells);
    if (rc) return rc;
    CK(cudaMemsetAsync(S.bin_first, 0xff, (size_t)h->g.cells * sizeof(int), h->stream));
    return LBM_OK;
}

// arrays only the comparison variants need
int ensure_comparison_arrays(lbm *h)
{
    int rc;
    if (h->opt_interp == 1)
        for (PrepSet &S : h->set) if (!S.inv && (rc = dmalloc(h, &S.inv, (size_t)h->nm_cap))) return rc;
    if (h->opt_moments == 1 && !h->d_box && (rc = dmalloc(h, &h->d_box, (size_t)6 * (size_t)h->nb_cap))) return rc;
    if (!fused_path(h))
        for (PrepSet &S : h->set) {
            // s g per marker; the round-1 sweep also reads per-marker weight tables.  A set prepared without them is stale.
            const size_t c = (size_t)h->nm_cap;
            if (!S.ms.sg) { if ((rc = dmalloc(h, &S.ms.sg, c))) return rc; S.step = -1; }
            if (h->opt_spread == 0 && !S.ms.wx) {
                if ((rc = dmalloc(h, &S.ms.wx, c))) return rc;
                if ((rc = dmalloc(h, &S.ms.wyz, 16 * c))) return rc;
                S.step = -1;
            }
        }
    return LBM_OK;
}

// ---- remove what the preparations registered in the dense maps (outside any graph) -------------
int flush_set(lbm *h, PrepSet &S)
{
    S.step = -1; S.stage = 0;
    if (!S.dirty) return LBM_OK;
    k_clear_prev<<<LIST_GRID, 256, 0, h->stream>>>(sorted_keys(h, S), &S.scal->n_prev, S.bin_first, S.amask, S.words,
                                                    &S.scal->n_words, S.chunk_of, S.ct.slot, &S.scal->n_chunks,
                                                    h->chunk_cap, S.tt.mask, S.tt.slot, &S.scal->n_tiles, h->tile_cap,
                                                    S.ovf_slot, &S.scal->n_ovf, OVF_CAP, (int)h->tile_slots);
    CK(cudaMemsetAsync(S.scal, 0, sizeof(SetScalars), h->stream));
    CK(cudaGetLastError());
    h->launches += 1;
    S.dirty = false;
    return LBM_OK;
}

int flush_ibm(lbm *h)
{
    for (PrepSet &S : h->set) {
        int rc = flush_set(h, S);
        if (rc) return rc;
    }
    h->force_valid = false;
    h->last_set = -1;
    return LBM_OK;
}

// ---- the fused MDF kernels for a tile edge and a lattice ---------------------------------------------
struct MdfKernels {
    void (*tiles)(const MdfArgs, int *, int, int);
    void (*pairs)(const MdfArgs, int *, int);
    void (*plan)(const MdfArgs);
    void (*persistent)(const MdfArgs, const float *, const PlaneOffsets, int *, unsigned *, int, int, const WordsArgs);
};

// How many (tile, footprint coordinate) candidates a cell can have per axis: two unless a 4-cell span can wrap
// onto its own tile or meet a third, narrow one (tiny or odd-sized periodic lattices); single-row and two-row
// tiles meet up to four tiles in y and z.
MdfKernels mdf_kernels(const lbm *h)
{
    const Geom &g = h->g;
    const bool two_x = g.wallx || g.nx >= CHUNK_ENT_MAX;
    const bool two_yz = (g.wally || g.ny % TILE_R == 0) && (g.wallz || g.nz % TILE_R == 0);
    switch (h->tr) {
        case 1:
            if (two_x) return MdfKernels{k_mdf_tiles<1>, k_mdf_pairs<1>, k_collect_plan<1, 2, 4>, k_mdf_persistent<1>};
            return MdfKernels{k_mdf_tiles<1>, k_mdf_pairs<1>, k_collect_plan<1, 4, 4>, k_mdf_persistent<1>};
        case 2:
            if (two_x) return MdfKernels{k_mdf_tiles<2>, k_mdf_pairs<2>, k_collect_plan<2, 2, 4>, k_mdf_persistent<2>};
            return MdfKernels{k_mdf_tiles<2>, k_mdf_pairs<2>, k_collect_plan<2, 4, 4>, k_mdf_persistent<2>};
        default:
            if (two_x && two_yz) return MdfKernels{k_mdf_tiles<4>, k_mdf_pairs<4>, k_collect_plan<4, 2, 2>, k_mdf_persistent<4>};
            return MdfKernels{k_mdf_tiles<4>, k_mdf_pairs<4>, k_collect_plan<4, 4, 4>, k_mdf_persistent<4>};
    }
}

constexpr int MDFP_BLOCKS_PER_SM = 1;   // the persistent kernel leaves room for the bulk stream-collide beside it

int mdf_launch_geometry(lbm *h)
{
    const MdfKernels K = mdf_kernels(h);
    const size_t smem_t = (size_t)MDF_WARPS * h->mdf_wsmem, smem_p = (size_t)MDFP_WARPS * h->mdf_wsmem;
    // The shared-memory cap is an attribute of the KERNEL, device-wide, shared by every handle of the process (and by
    // every host thread): it is set to what the widest window needs (CHUNK_ENT_MAX entries), never to this handle's own
    // size -- a handle on a lattice with a narrower window would otherwise lower the cap under the graphs another
    // handle has still to build.
    const ChunkGeom widest{1, CHUNK_ENT_MAX};
    const size_t wmax = mdf_warp_smem(h->tr, widest);
    CK(cudaFuncSetAttribute((const void *)K.tiles, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(MDF_WARPS * wmax)));
    CK(cudaFuncSetAttribute((const void *)K.persistent, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(MDFP_WARPS * wmax)));
    int per_sm = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, K.tiles, MDF_WARPS * 32, smem_t));
    if (h->opt_mdf_blocks > 0) per_sm = std::min(per_sm, h->opt_mdf_blocks);
    h->mdf_grid = std::max(1, per_sm) * h->sms;
    const size_t smem_2 = mdf_pair_smem(h->tr, h->cg);
    CK(cudaFuncSetAttribute((const void *)K.pairs, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mdf_pair_smem(h->tr, widest)));
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, K.pairs, 64, smem_2));
    if (h->opt_mdf_blocks > 0) per_sm = std::min(per_sm, h->opt_mdf_blocks);
    h->mdf2_grid = std::max(1, per_sm) * h->sms;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, K.persistent, MDFP_WARPS * 32, smem_p));
    if (per_sm < 1) return fail(LBM_ECUDA, "the persistent MDF kernel does not fit on an SM (%zu bytes of shared memory)", smem_p);
    h->mdfp_grid = std::min(per_sm, h->opt_mdf_blocks > 0 ? h->opt_mdf_blocks : MDFP_BLOCKS_PER_SM) * h->sms;
    return LBM_OK;
}

MdfArgs mdf_args(const lbm *h, const PrepSet &S)
{
    MdfArgs a{};
    a.g = h->g; a.cg = h->cg; a.tg = h->tg;
    a.tile_rec = S.tt.rec; a.tile_slot = S.tt.slot; a.tile_mask = S.tt.mask; a.tile_id = S.tt.id; a.tile_ohdr = S.tt.ohdr; a.tile_orec = S.tt.orec;
    a.tile_order = S.tile_order; a.n_tiles = &S.scal->n_tiles; a.tile_cap = h->tile_cap;
    a.fdst = S.fdst; a.cell_run = S.cell_run; a.n_felem = &S.scal->n_felem;
    a.fs = S.ms.fs; a.uk = S.ms.uk; a.du = S.ms.du;
    a.U = h->U; a.G = h->G; a.F = h->F;
    a.cells = S.cells; a.n_cells = &S.scal->n_cells;
    return a;
}

// ---- (re)build the device copies of the markers -------------------------------------------------
int upload_markers(lbm *h)
{
    if (!h->markers_stale) return LBM_OK;
    int rc = flush_ibm(h);
    if (rc) return rc;
    CK(cudaStreamSynchronize(h->stream));
    drop_graphs(h);
    const int n = (int)h->h_area.size();
    const int nb = (int)h->bodies.size();
    const int tr = effective_tr(h);
    if (n > h->nm_cap || nb > h->nb_cap || tr != h->tr || h->realloc_tables) {
        free_markers_dev(h);
        h->realloc_tables = false;
        h->tr = tr;
        h->tg = tile_geom(h->g.ny, h->g.nz, tr);
        h->tile_slots = (size_t)h->cg.nbx * h->tg.nty * h->tg.ntz;
        const size_t c = (size_t)n;
        if ((rc = dmalloc(h, &h->d_qs, c))) return rc;
        if ((rc = dmalloc(h, &h->d_vb, c))) return rc;
        if ((rc = dmalloc(h, &h->d_body, c))) return rc;
        // every chunk that can exist gets a table entry (one per marker, one per (row, block) slot, CHUNK_ID_MAX);
        // F has room for every tile that can exist up to 12 GB, beyond that the capacity is capped and an
        // overflow is flagged on the device (LBM_ENOMEM at lbm_sync)
        const size_t ccap = std::max((size_t)1, std::min(std::min(c, h->chunk_slots), (size_t)CHUNK_ID_MAX));
        const size_t tile_elems = (size_t)((tr + 3) * (tr + 3)) * (size_t)h->cg.ent;
        size_t tcap = std::max((size_t)1, std::min(std::min(c, h->tile_slots), ((size_t)12 << 30) / (tile_elems * sizeof(float4))));
        if (h->opt_tile_cap > 0) tcap = std::max((size_t)1, std::min(tcap, (size_t)h->opt_tile_cap));   // LBM_OPT_TILE_CAP
        // active cells: a chunk marks the whole x span between the windows of its first and its last marker in 16 rows,
        // cells between two far-apart markers included: one marker alone activates 64 cells, two markers of a chunk up to
        // CHUNK_ENT_MAX x 16, i.e. at most 8 x CHUNK_ENT_MAX cells per marker
        h->cells_cap = std::min((size_t)(8 * CHUNK_ENT_MAX) * c, (size_t)h->g.cells);
        h->headbits_cap = c / 32 + 16;
        for (PrepSet &S : h->set) {
            for (int a = 0; a < 2; ++a) {
                if ((rc = dmalloc(h, &S.keys[a], c))) return rc;
                if ((rc = dmalloc(h, &S.vals[a], c))) return rc;
            }
            if ((rc = dmalloc(h, &S.ms.fs, c))) return rc;
            if ((rc = dmalloc(h, &S.ms.uk, c))) return rc;
            if ((rc = dmalloc(h, &S.ms.du, c))) return rc;      // wx, wyz, sg: comparison paths only (ensure_comparison_arrays)
            if ((rc = dmalloc(h, &S.ct.first, (size_t)ccap))) return rc;
            if ((rc = dmalloc(h, &S.ct.end, (size_t)ccap))) return rc;
            if ((rc = dmalloc(h, &S.ct.slot, (size_t)ccap))) return rc;
            if ((rc = dmalloc(h, &S.tt.slot, tcap))) return rc;
            if ((rc = dmalloc(h, &S.tt.ohdr, tcap))) return rc;
            if ((rc = dmalloc(h, &S.tt.orec, tcap * (size_t)(tr * tr)))) return rc;
            if ((rc = dmalloc(h, &S.tt.rec, tcap * (size_t)(tr * tr)))) return rc;
            if ((rc = dmalloc(h, &S.tile_order, tcap))) return rc;
            if ((rc = dmalloc(h, &S.ovf_slot, (size_t)OVF_CAP))) return rc;
            if ((rc = dmalloc(h, &S.fdst, tcap * tile_elems))) return rc;
            if ((rc = dmalloc(h, &S.cell_run, h->cells_cap))) return rc;
            if ((rc = dmalloc(h, &S.tt.mask, h->tile_slots))) return rc;
            if ((rc = dmalloc(h, &S.tt.id, h->tile_slots))) return rc;
            CK(cudaMemsetAsync(S.tt.mask, 0, h->tile_slots * sizeof(unsigned), h->stream));
            if ((rc = dmalloc(h, &S.cells, h->cells_cap))) return rc;
            if ((rc = dmalloc(h, &S.headbits, h->headbits_cap))) return rc;
        }
        if ((rc = dmalloc(h, &h->F, tcap * tile_elems))) return rc;
        h->chunk_cap = (int)ccap; h->tile_cap = (int)tcap;
        // launch geometry of the fused tile pass and of the persistent MDF kernel for (tr, cg)
        h->mdf_wsmem = mdf_warp_smem(tr, h->cg);
        if ((rc = mdf_launch_geometry(h))) return rc;
        for (int i = 0; i < N_SETS; ++i) if ((rc = dmalloc(h, &h->d_total[i], (size_t)RADIX))) return rc;
        if ((rc = dmalloc(h, &h->d_defs, (size_t)nb))) return rc;
        for (PrepSet &S : h->set) if ((rc = dmalloc(h, &S.tabs, (size_t)nb))) return rc;
        h->nm_cap = n; h->nb_cap = nb;
    }
    h->nm = n;
    // sort geometry
    int ipw = ((n / (148 * 32)) + 31) / 32 * 32;
    if (ipw < 64) ipw = 64;
    if (ipw > 2048) ipw = 2048;
    const int tiles = n > 0 ? (n + ipw - 1) / ipw : 0;
    if (tiles > h->sort_tiles) {
        for (int i = 0; i < N_SETS; ++i) {
            dfree(h, h->d_hist[i], (size_t)RADIX * (size_t)h->sort_tiles);
            if ((rc = dmalloc(h, &h->d_hist[i], (size_t)RADIX * (size_t)tiles))) return rc;
        }
    }
    h->sort_ipw = ipw; h->sort_tiles = tiles;
    int bits = 1;
    while (bits < 32 && ((long long)1 << bits) < h->g.cells) ++bits;
    h->sort_passes = (bits + 7) / 8;
    if (n == 0) { h->markers_stale = false; return LBM_OK; }

    // body tables; rest positions relative to the body centre, formed in fp64
    std::vector<BodyDef> &defs = h->h_defs;
    defs.assign((size_t)nb, BodyDef{});
    std::vector<float4> qs((size_t)n), vb((size_t)n);
    for (int b = 0; b < nb; ++b) {
        const HostBody &B = h->bodies[(size_t)b];
        BodyDef d{};
        d.omega = B.omega; d.ax = B.axis[0]; d.ay = B.axis[1]; d.az = B.axis[2];
        for (int a = 0; a < 3; ++a) {
            const double fl = std::floor(B.center[a]);
            d.ci[a] = (int)fl;
            d.cf[a] = (float)(B.center[a] - fl);
            if (d.cf[a] >= 1.0f) { d.cf[a] = 0.0f; d.ci[a] += 1; }
        }
        defs[(size_t)b] = d;
        for (long long k = B.first; k < B.first + B.count; ++k) {
            const size_t i = (size_t)k;
            float bits;
            std::memcpy(&bits, &b, sizeof bits);
            qs[i] = make_float4((float)((double)h->h_pos[3 * i] - B.center[0]), (float)((double)h->h_pos[3 * i + 1] - B.center[1]),
                                (float)((double)h->h_pos[3 * i + 2] - B.center[2]), h->h_area[i]);
            vb[i] = make_float4(h->h_vel[3 * i], h->h_vel[3 * i + 1], h->h_vel[3 * i + 2], bits);
        }
    }
    CK(cudaMemcpyAsync(h->d_qs, qs.data(), sizeof(float4) * (size_t)n, cudaMemcpyHostToDevice, h->stream));
    CK(cudaMemcpyAsync(h->d_vb, vb.data(), sizeof(float4) * (size_t)n, cudaMemcpyHostToDevice, h->stream));
    CK(cudaMemcpyAsync(h->d_body, h->h_body.data(), sizeof(int) * (size_t)n, cudaMemcpyHostToDevice, h->stream));
    CK(cudaMemcpyAsync(h->d_defs, defs.data(), sizeof(BodyDef) * (size_t)nb, cudaMemcpyHostToDevice, h->stream));
    CK(cudaStreamSynchronize(h->stream));   // staging vectors die here
    h->markers_stale = false;
    return LBM_OK;
}

// ---- launch helpers (plain launches on stream s; also what graph capture records) --------------

// a1-a3 for the time step (device step counter + step_offset) into marker set S.  parts: bit 0 = first half
// (kinematics tables, keys, sort), bit 1 = second half (gather, chunks, tiles, active cells, collect plan).
enum { PREP_SORT = 1, PREP_BINS = 2, PREP_ALL = 3 };
int enqueue_prep(lbm *h, cudaStream_t s, PrepSet &S, int step_offset, int *n_kernels, PhaseTimer *pt, int parts = PREP_ALL,
                 bool advance_step = false)
{
    const Geom &g = h->g;
    const int n = h->nm;
    const int mb = (n + 255) / 256;
    SetScalars *sc = S.scal;
    unsigned *skey = S.keys[h->sort_passes & 1];
    int *perm = S.vals[h->sort_passes & 1];
    MarkerIn mi{h->d_qs, h->d_vb, h->d_body, n};
    int nk = 0;
    const int lg = list_grid(h);

    if (parts & PREP_SORT) {
    if (pt) pt->mark(PH_KEYS, s);
    k_clear_prev<<<lg, 256, 0, s>>>(skey, &sc->n_prev, S.bin_first, S.amask, S.words, &sc->n_words, S.chunk_of,
                                           S.ct.slot, &sc->n_chunks, h->chunk_cap, S.tt.mask, S.tt.slot, &sc->n_tiles, h->tile_cap,
                                           S.ovf_slot, &sc->n_ovf, OVF_CAP, (int)h->tile_slots);
    const int nb = (int)h->bodies.size();
    k_kinematics<<<(std::max(nb, N_STEP_COUNTERS) + 127) / 128, 128, 0, s>>>(h->d_defs, S.tabs, nb, &h->scal->step_ctr,
                                                                              step_offset, &sc->n_words, N_STEP_COUNTERS);
    k_marker_keys<<<mb, 256, 0, s>>>(mi, h->d_defs, S.tabs, g, S.keys[0], &h->scal->status,
                                     advance_step ? &h->scal->step_ctr : nullptr);
    nk += 3;
    if (pt) pt->mark(PH_SORT, s);
    if (n <= SORT_SMALL_MAX) {
        // small marker sets: every pass in one single-block kernel (same result, 3 launches instead of 3 per pass)
        k_radix_sort_small<<<1, SORT_SMALL_BLOCK, 0, s>>>(S.keys[0], S.keys[1], S.vals[0], S.vals[1], n, h->sort_passes);
        ++nk;
    } else {
        const int sb = (h->sort_tiles + SORT_WARPS - 1) / SORT_WARPS;
        const int si = (int)(&S - h->set);
        int *hist = h->d_hist[si], *total = h->d_total[si];
        for (int p = 0; p < h->sort_passes; ++p) {
            const unsigned *kin = S.keys[p & 1];
            unsigned *kout = S.keys[(p + 1) & 1];
            const int *vin = p == 0 ? nullptr : S.vals[p & 1];
            int *vout = S.vals[(p + 1) & 1];
            k_radix_hist<<<sb, SORT_BLOCK, 0, s>>>(kin, n, h->sort_ipw, h->sort_tiles, 8 * p, hist);
            k_radix_scan<<<RADIX, SORT_BLOCK, 0, s>>>(hist, h->sort_tiles, total);
            k_radix_scatter<<<sb, SORT_BLOCK, 0, s>>>(kin, vin, kout, vout, n, h->sort_ipw, h->sort_tiles, 8 * p, hist, total);
            nk += 3;
        }
    }
    trace_mark(h, s, step_offset == 2 ? "prep2.sort" : "prep.sort");
    }
    if (!(parts & PREP_BINS)) { CK(cudaGetLastError()); *n_kernels += nk; return LBM_OK; }
    if (pt) pt->mark(PH_BINS, s);
    k_marker_gather<<<mb, 256, 0, s>>>(mi, h->d_defs, S.tabs, g, perm, S.ms);
    ++nk;
    if (h->opt_interp == 1) { k_invert_perm<<<mb, 256, 0, s>>>(perm, n, S.inv); ++nk; }
    if (h->opt_spread == 0) {
        k_chunk_heads<<<(n + 32 + 255) / 256, 256, 0, s>>>(skey, n, g, h->cg, S.headbits);
        k_chunks<<<mb, 256, 0, s>>>(skey, n, g, h->cg, S.headbits, S.ct, h->chunk_cap, &sc->n_chunks, &sc->n_entries,
                                    S.chunk_of, &h->scal->status);
        k_chunk_publish<<<lg, 256, 0, s>>>(g, h->cg, S.ct, &sc->n_chunks, h->chunk_cap, S.chunk_of, S.amask);
        k_tiles<<<lg, 256, 0, s>>>(g, h->cg, h->tg, S.ct, &sc->n_chunks, h->chunk_cap, S.chunk_of, S.tt, h->tile_cap,
                                          &sc->n_tiles, S.ovf_slot, OVF_CAP, &sc->n_ovf, &h->scal->status);
        k_tile_fill<<<lg, 256, 0, s>>>(g, h->cg, h->tg, S.ct, &sc->n_chunks, h->chunk_cap, S.tt);
        k_tile_count<<<lg, 256, 0, s>>>(S.tt, h->tr * h->tr, &sc->n_tiles, h->tile_cap, sc->bucket);
        k_tile_place<<<lg, 256, 0, s>>>(S.tt, h->tr * h->tr, &sc->n_tiles, h->tile_cap, sc->bucket, S.tile_order);
        nk += 7;
    } else {
        k_bins<<<mb, 256, 0, s>>>(skey, n, g, S.bin_first, S.amask);
        ++nk;
    }
    k_compact_words<<<(int)std::min<size_t>(LIST_GRID, (h->n_mask_words + 255) / 256), 256, 0, s>>>(S.amask, (int)h->n_mask_words, S.words, &sc->n_words);
    k_active_cells<<<lg, 256, 0, s>>>(g, S.amask, S.words, &sc->n_words, S.cells, &sc->n_cells);
    if (h->opt_spread == 0) {
        // collect plan: which footprint elements every active cell adds up, and where the tile pass puts them
        const int elems = (h->tr + 3) * (h->tr + 3) * h->cg.ent;
        k_fill_tiles<<<lg, 256, 0, s>>>(S.fdst, &sc->n_tiles, h->tile_cap, elems);
        mdf_kernels(h).plan<<<lg, 256, 0, s>>>(mdf_args(h, S));
        nk += 2;
    }
    k_set_scalars<<<1, 1, 0, s>>>(&h->scal->step_ctr, 0, &sc->n_prev, n, 2);
    nk += 3;
    CK(cudaGetLastError());
    *n_kernels += nk;
    return LBM_OK;
}

CollisionConst collision_const(const lbm *h);

// a4-a7: moments on the active cells of set S, then the MDF loop; leaves G on the active cells.
// words_dst != NULL (persistent kernel only): the kernel also runs the stream-collide of the cells inside the stencils
// into that buffer once G is complete.
int enqueue_mdf(lbm *h, cudaStream_t s, PrepSet &S, const float *src, int mdf_iters, int *n_kernels, PhaseTimer *pt,
                float *words_dst = nullptr)
{
    const Geom &g = h->g;
    const int n = h->nm;
    SetScalars *sc = S.scal;
    const unsigned *skey = sorted_keys(h, S);
    int nk = 0;
    const bool fused = fused_path(h);
    const int lg = list_grid(h);
    const MdfKernels K = mdf_kernels(h);
    const MdfArgs ma = mdf_args(h, S);
    const int wsmem = (int)h->mdf_wsmem;
    if (use_persistent(h)) {
        // a4 + the whole loop in one kernel: grid-wide barriers instead of 2 N + 1 dependent launches
        WordsArgs wa{};
        wa.dst = words_dst; wa.cc = collision_const(h); wa.amask = S.amask; wa.words = S.words; wa.n_words = &sc->n_words;
        wa.enabled = words_dst ? 1 : 0;
        K.persistent<<<h->mdfp_grid, MDFP_WARPS * 32, (size_t)MDFP_WARPS * h->mdf_wsmem, s>>>(
            ma, src, h->po, sc->cursor, &sc->gbar, mdf_iters, wsmem, wa);
        if (!words_dst) trace_mark(h, s, "mdf_persistent");   // with the words pass inside: marked by the caller, off this stream
        CK(cudaGetLastError());
        *n_kernels += 1;
        return LBM_OK;
    }
    if (pt) pt->mark(PH_MOMENTS, s);
    if (h->opt_moments == 1) {
        // the paper's box strategy: U on the bounding box of every body
        const int nb = (int)h->bodies.size();
        MarkerIn mi{h->d_qs, h->d_vb, h->d_body, n};
        k_reset_boxes<<<(nb + 127) / 128, 128, 0, s>>>(h->d_box, nb);
        k_body_boxes<<<(n + 255) / 256, 256, 0, s>>>(mi, h->d_defs, S.tabs, h->d_box);   // the set's own tables
        k_moments_box<<<dim3(64, nb), 256, 0, s>>>(src, g, h->d_box, h->U);
        nk += 3;
    } else if (h->opt_moments == 2) {
        // the paper's kernel strategy: a block per Lagrangian point, duplicates included
        k_moments_per_marker<<<n, 64, 0, s>>>(src, g, skey, n, h->U);
        ++nk;
    } else {
        k_moments_active<<<h->moments_grid, 256, 0, s>>>(src, g, h->po, S.cells, &sc->n_cells, h->U);
        ++nk;
    }
    trace_mark(h, s, "moments");
    for (int m = 0; m < mdf_iters; ++m) {
        const bool last = (m == mdf_iters - 1);
        if (pt) pt->mark(PH_INTERP, s);
        if (fused) {
            // product path: interpolate + correct + sweep in one tile pass, then the collect
            if (tile_warps(h) == 2)
                K.pairs<<<h->mdf2_grid, 64, mdf_pair_smem(h->tr, h->cg), s>>>(ma, &sc->cursor[m], last ? 1 : 0);
            else
                K.tiles<<<h->mdf_grid, MDF_WARPS * 32, (size_t)MDF_WARPS * h->mdf_wsmem, s>>>(ma, &sc->cursor[m], last ? 1 : 0, wsmem);
            trace_mark(h, s, "tiles", m);
            if (pt) pt->mark(PH_SPREAD, s);
            k_mdf_collect<<<lg, 256, 0, s>>>(ma, last ? 1 : 0);
            trace_mark(h, s, "collect", m);
            nk += 2;
            continue;
        }
        if (h->opt_interp == 1) k_interp_caller_order<<<(n + 127) / 128, 128, 0, s>>>(skey, S.inv, n, g, h->U, S.ms);
        else if (h->opt_interp == 2) k_interp_warp_per_marker<<<(int)(((long long)n * 32 + 255) / 256), 256, 0, s>>>(skey, n, g, h->U, S.ms);
        else if (h->opt_interp == 3 && h->opt_spread == 0)
            k_interp_chunks<<<148 * 8, ICHUNK_WARPS * 32, 0, s>>>(skey, g, h->cg, S.ct, &sc->n_chunks, h->chunk_cap, &sc->icursor[m],
                                                                  h->U, S.ms);
        else k_interp_correct<<<(n + 127) / 128, 128, 0, s>>>(skey, n, g, h->U, S.ms);
        ++nk;
        if (pt) pt->mark(PH_SPREAD, s);
        if (h->opt_spread == 0) {
            // the round-1 pipeline (LBM_OPT_FUSED = 0): separate interpolation kernel, TMA-fed warp-per-tile sweep
            k_spread_tiles<<<h->rows_grid, TILE_WARPS * 32, spread_tiles_smem(h->cg), s>>>(
                h->cg, S.tt.rec, S.tt.slot, S.tt.mask, &sc->n_tiles, h->tile_cap, &sc->cursor[m], S.tile_order, S.ms.wx,
                S.ms.wyz, last ? S.ms.du : S.ms.sg, S.fdst, h->F, (int)spread_warp_smem(h->cg));
            k_mdf_collect<<<lg, 256, 0, s>>>(ma, last ? 1 : 0);
            nk += 2;
        } else if (h->opt_spread == 2) {
            if (last)
                k_spread_gather<true><<<lg, 256, 0, s>>>(skey, n, g, S.bin_first, S.amask, S.words, &sc->n_words,
                                                                 S.ms.fs, S.ms.du, h->G);
            else
                k_spread_gather<false><<<lg, 256, 0, s>>>(skey, n, g, S.bin_first, S.amask, S.words, &sc->n_words,
                                                                  S.ms.fs, S.ms.sg, h->U);
            ++nk;
        } else {
            // global atomics: thread per marker (1) or the paper's block of 5^3 threads per marker (3)
            if (last) { k_zero_active<<<lg, 256, 0, s>>>(g, S.amask, S.words, &sc->n_words, h->G); ++nk; }
            const float4 *v = last ? S.ms.du : S.ms.sg;
            float4 *field = last ? h->G : h->U;
            if (h->opt_spread == 3) k_spread_block125<<<n, 125, 0, s>>>(skey, n, g, S.ms.fs, v, field);
            else k_spread_atomic<<<(n + 127) / 128, 128, 0, s>>>(skey, n, g, S.ms.fs, v, field);
            ++nk;
        }
    }
    CK(cudaGetLastError());
    *n_kernels += nk;
    return LBM_OK;
}

CollisionConst collision_const(const lbm *h)
{
    CollisionConst cc = h->cc;
    cc.shift_forcing = h->opt_forcing;
    return cc;
}

// a8 in one pass over the whole lattice: mode LBM_PURE, LBM_FUSED (mask + G) or LBM_BULK (skip active cells)
int enqueue_lbm_pass(lbm *h, cudaStream_t s, const float *src, float *dst, int mode, const unsigned *amask)
{
    const Geom &g = h->g;
    const CollisionConst cc = collision_const(h);
    const bool vec = (h->opt_lbm_kernel == 2) && (g.nx % 4 == 0) && (mode == LBM_PURE || mode == LBM_FUSED);
    if (vec) {
        const int nx4 = g.nx / 4;
        int bx = 1;
        while (bx < nx4 && bx < 64) bx <<= 1;
        dim3 b(bx, 256 / bx, 1);
        dim3 gr((nx4 + b.x - 1) / b.x, (g.ny + b.y - 1) / b.y, g.nz);
        if (mode == LBM_FUSED) k_stream_collide_vec4<true><<<gr, b, 0, s>>>(src, dst, g, cc, amask, h->G);
        else k_stream_collide_vec4<false><<<gr, b, 0, s>>>(src, dst, g, cc, nullptr, nullptr);
    } else {
        const dim3 b = cell_block(g);
        const dim3 gr = cell_grid(g, b);
        if (mode == LBM_FUSED) k_stream_collide_scalar<LBM_FUSED, 256, 5><<<gr, b, 0, s>>>(src, dst, g, cc, h->po, amask, h->G);
        else if (mode == LBM_BULK && bulk_stream(h)) k_stream_collide_scalar<LBM_BULK, 256, 5, true><<<gr, b, 0, s>>>(src, dst, g, cc, h->po, amask, nullptr);
        else if (mode == LBM_BULK) k_stream_collide_scalar<LBM_BULK, 256, 5><<<gr, b, 0, s>>>(src, dst, g, cc, h->po, amask, nullptr);
        else k_stream_collide_scalar<LBM_PURE, 256, 5><<<gr, b, 0, s>>>(src, dst, g, cc, h->po, nullptr, nullptr);
    }
    CK(cudaGetLastError());
    return LBM_OK;
}

int enqueue_lbm_active(lbm *h, cudaStream_t s, const float *src, float *dst, PrepSet &S)
{
    k_stream_collide_words<<<h->words_grid, 256, 0, s>>>(src, dst, h->g, collision_const(h), h->po, S.amask, S.words,
                                                      &S.scal->n_words, h->G, &h->scal->step_ctr);
    CK(cudaGetLastError());
    return LBM_OK;
}

// ---- one time step, serial on stream s ----------------------------------------------------------
// prep: 0 = set S is already prepared for this step; 1 = prepare it first.
int enqueue_step_serial(lbm *h, cudaStream_t s, int parity, PrepSet *S, bool prep, int mdf_iters, int *n_kernels,
                        PhaseTimer *pt = nullptr)
{
    const float *src = h->f[parity];
    float *dst = h->f[parity ^ 1];
    int nk = 0, rc;
    if (S) {
        if (prep && (rc = enqueue_prep(h, s, *S, 0, &nk, pt))) return rc;
        if ((rc = enqueue_mdf(h, s, *S, src, mdf_iters, &nk, pt))) return rc;
        if (overlap_mode(h) == 1) {
            if (pt) pt->mark(PH_LBM, s);
            if ((rc = enqueue_lbm_pass(h, s, src, dst, LBM_BULK, S->amask))) return rc;
            if (pt) pt->mark(PH_LBM_ACTIVE, s);
            if ((rc = enqueue_lbm_active(h, s, src, dst, *S))) return rc;     // also advances the step counter
            nk += 2;
        } else {
            if (pt) pt->mark(PH_LBM, s);
            if ((rc = enqueue_lbm_pass(h, s, src, dst, LBM_FUSED, S->amask))) return rc;
            k_set_scalars<<<1, 1, 0, s>>>(&h->scal->step_ctr, 0, nullptr, 0, 4);
            nk += 2;
        }
    } else {
        if (pt) pt->mark(PH_LBM, s);
        if ((rc = enqueue_lbm_pass(h, s, src, dst, LBM_PURE, nullptr))) return rc;
        ++nk;
    }
    if (pt) pt->mark(-1, s);
    CK(cudaGetLastError());
    *n_kernels = nk;
    return LBM_OK;
}

// ---- one time step as concurrent branches (captured into a graph) ------------------------------------
//   main (high priority): moments + MDF loop on set S          -> G
//   bulk (low priority) : stream-collide of every cell outside S's active mask (needs no G); layout 1 only
//   prep                : binning of step n + 1 into set N: its second half if the first was done during step n - 1
//                         (n_has_sort), else all of it
//   prep2               : first half of the binning of step n + 2 into set N2 (pipeline depth 2 only, N2 != NULL)
//   join, then the stream-collide of the active cells with G (layout 2: of all cells), then step counter + 1.
int enqueue_step_overlapped(lbm *h, int parity, PrepSet &S, PrepSet &N, PrepSet *N2, bool n_has_sort, int mdf_iters,
                            int *n_kernels)
{
    const float *src = h->f[parity];
    float *dst = h->f[parity ^ 1];
    cudaStream_t s = h->cap_stream;
    int nk = 0, rc;
    const bool split = overlap_mode(h) == 1;    // 1: bulk stream-collide beside the MDF loop; 2: one fused pass after it
    trace_mark(h, s, "fork");
    CK(cudaEventRecord(h->ev_fork, s));
    const bool pdl = split && use_persistent(h);
    if (split && !pdl) CK(cudaStreamWaitEvent(h->cap_bulk, h->ev_fork, 0));
    CK(cudaStreamWaitEvent(h->cap_prep, h->ev_fork, 0));
    if (N2) CK(cudaStreamWaitEvent(h->cap_prep2, h->ev_fork, 0));
    if (split && !pdl) {
        if ((rc = enqueue_lbm_pass(h, h->cap_bulk, src, dst, LBM_BULK, S.amask))) return rc;
        trace_mark(h, h->cap_bulk, "bulk");
        ++nk;
    }
    // with the persistent MDF kernel the cells inside the stencils are updated by that kernel itself (it needs G, not
    // the bulk pass: the two passes write disjoint cells); the step counter then advances in a kernel of its own
    const bool fold = split && use_persistent(h);
    if ((rc = enqueue_mdf(h, s, S, src, mdf_iters, &nk, nullptr, fold ? dst : nullptr))) return rc;
    if (pdl) {
        // the bulk pass as a programmatic dependent of the persistent kernel: it starts when every block of that
        // grid is resident (griddepcontrol.launch_dependents at its top), not before
        CK(cudaEventRecord(h->ev_mdf, s));
        if (h->opt_trace) {
            // the trace event of the persistent kernel goes to a side stream: an event node between the two kernels
            // would turn the programmatic edge into a full dependency
            CK(cudaStreamWaitEvent(h->cap_bulk, h->ev_mdf, 0));
            trace_mark(h, h->cap_bulk, "mdf_persistent");
            CK(cudaEventRecord(h->ev_bulk, h->cap_bulk));
        }
        const dim3 b = cell_block(h->g);
        const dim3 gr = cell_grid(h->g, b);
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = gr; cfg.blockDim = b; cfg.dynamicSmemBytes = 0; cfg.stream = s;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        const CollisionConst cc = collision_const(h);
        if (bulk_stream(h))
            CK(cudaLaunchKernelEx(&cfg, k_stream_collide_scalar<LBM_BULK, 256, 5, true>, src, dst, h->g, cc, h->po,
                                  (const unsigned *)S.amask, (const float4 *)nullptr));
        else
            CK(cudaLaunchKernelEx(&cfg, k_stream_collide_scalar<LBM_BULK, 256, 5>, src, dst, h->g, cc, h->po,
                                  (const unsigned *)S.amask, (const float4 *)nullptr));
        trace_mark(h, s, "bulk");
        ++nk;
    }
    if ((rc = enqueue_prep(h, h->cap_prep, N, 1, &nk, nullptr, n_has_sort ? PREP_BINS : PREP_ALL))) return rc;
    trace_mark(h, h->cap_prep, "prep");
    // steady state of the depth-2 pipeline with the persistent kernel: the only reader of the step counter in this
    // graph is the k_kinematics of the prep2 chain, and the counter advances right behind it in that chain
    const bool ctr_in_prep2 = fold && N2 && n_has_sort;
    if (N2) {
        if ((rc = enqueue_prep(h, h->cap_prep2, *N2, 2, &nk, nullptr, PREP_SORT, ctr_in_prep2))) return rc;
        trace_mark(h, h->cap_prep2, "prep2");
    }
    if (split && !pdl) CK(cudaEventRecord(h->ev_bulk, h->cap_bulk));
    CK(cudaEventRecord(h->ev_prep, h->cap_prep));
    if (N2) CK(cudaEventRecord(h->ev_prep2, h->cap_prep2));
    if (split && !pdl) CK(cudaStreamWaitEvent(s, h->ev_bulk, 0));
    if (pdl) CK(cudaStreamWaitEvent(s, h->ev_mdf, 0));
    if (pdl && h->opt_trace) CK(cudaStreamWaitEvent(s, h->ev_bulk, 0));
    CK(cudaStreamWaitEvent(s, h->ev_prep, 0));
    if (N2) CK(cudaStreamWaitEvent(s, h->ev_prep2, 0));
    if (fold) {
        trace_mark(h, s, "join");
        if (!ctr_in_prep2) { k_set_scalars<<<1, 1, 0, s>>>(&h->scal->step_ctr, 0, nullptr, 0, 4); ++nk; }
    } else if (split) {
        trace_mark(h, s, "join");
        if ((rc = enqueue_lbm_active(h, s, src, dst, S))) return rc;           // also advances the step counter
        ++nk;
    } else {
        trace_mark(h, s, "join");
        if ((rc = enqueue_lbm_pass(h, s, src, dst, LBM_FUSED, S.amask))) return rc;
        k_set_scalars<<<1, 1, 0, s>>>(&h->scal->step_ctr, 0, nullptr, 0, 4);
        nk += 2;
    }
    trace_mark(h, s, "end");
    CK(cudaGetLastError());
    *n_kernels = nk;
    return LBM_OK;
}

// kind: 0 = pure LBM, 1 = serial IBM step that prepares its own set, 2 = overlapped IBM step
// pipe: for kind 2, bit 0 = the next step's set already holds its sorted keys, bit 1 = pipeline depth 2
int get_graph(lbm *h, int kind, int parity, int set, int mdf_iters, cudaGraphExec_t *exec, int *n_kernels, int pipe = 0)
{
    const long long key = ((long long)mdf_iters << 8) | ((long long)kind << 4) | (set << 1) | parity |
                          ((long long)h->opt_spread << 40) | ((long long)h->opt_forcing << 44) |
                          ((long long)h->opt_lbm_kernel << 48) | ((long long)h->opt_interp << 52) |
                          ((long long)overlap_mode(h) << 56) | ((long long)h->opt_moments << 58) |
                          ((long long)h->opt_fused << 60) | ((long long)h->tr << 16) | ((long long)use_persistent(h) << 20) |
                          ((long long)tile_warps(h) << 21) | ((long long)h->opt_trace << 23) | ((long long)pipe << 24) |
                          ((long long)h->opt_bulk_stream << 26);
    h->last_key = key;
    auto it = h->graphs.find(key);
    if (it != h->graphs.end()) { *exec = it->second.first; *n_kernels = it->second.second; return LBM_OK; }
    cudaGraph_t graph = nullptr;
    if (h->opt_trace && kind == 2) h->trace_cap = &h->traces[key];
    CK(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal));
    int nk = 0, rc;
    if (kind == 2)
        rc = enqueue_step_overlapped(h, parity, h->set[set], h->set[(set + 1) % N_SETS],
                                     (pipe & 2) ? &h->set[(set + 2) % N_SETS] : nullptr, (pipe & 1) != 0, mdf_iters, &nk);
    else rc = enqueue_step_serial(h, h->cap_stream, parity, kind ? &h->set[set] : nullptr, true, mdf_iters, &nk);
    cudaError_t e = cudaStreamEndCapture(h->cap_stream, &graph);
    h->trace_cap = nullptr;
    if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
    if (e != cudaSuccess) return fail(LBM_ECUDA, "graph capture failed: %s", cudaGetErrorString(e));
    if (kind == 2) {
        // node priorities: the lattice-wide bulk pass yields to every other kernel of the step, so that the short
        // IBM kernels are placed on the SMs as soon as bulk blocks retire instead of queueing behind the whole grid
        int lo = 0, hi = 0;
        cudaDeviceGetStreamPriorityRange(&lo, &hi);
        size_t nn = 0;
        e = cudaGraphGetNodes(graph, nullptr, &nn);
        std::vector<cudaGraphNode_t> nodes(nn);
        if (e == cudaSuccess) e = cudaGraphGetNodes(graph, nodes.data(), &nn);
        const void *bulk_fn = (const void *)k_stream_collide_scalar<LBM_BULK, 256, 5>;
        const void *bulk_cs_fn = (const void *)k_stream_collide_scalar<LBM_BULK, 256, 5, true>;
        for (size_t i = 0; i < nn && e == cudaSuccess; ++i) {
            cudaGraphNodeType ty;
            if (cudaGraphNodeGetType(nodes[i], &ty) != cudaSuccess || ty != cudaGraphNodeTypeKernel) continue;
            cudaKernelNodeParams kp{};
            if (cudaGraphKernelNodeGetParams(nodes[i], &kp) != cudaSuccess) continue;
            cudaLaunchAttributeValue v{};
            v.priority = (kp.func == bulk_fn || kp.func == bulk_cs_fn) ? lo : hi;
            e = cudaGraphKernelNodeSetAttribute(nodes[i], cudaLaunchAttributePriority, &v);
        }
        if (e != cudaSuccess) {
            cudaGraphDestroy(graph);
            return fail(LBM_ECUDA, "setting graph node priorities failed: %s", cudaGetErrorString(e));
        }
    }
    cudaGraphExec_t ex = nullptr;
    e = cudaGraphInstantiate(&ex, graph, kind == 2 ? cudaGraphInstantiateFlagUseNodePriority : 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) return fail(LBM_ECUDA, "graph instantiate failed: %s", cudaGetErrorString(e));
    h->graphs[key] = std::make_pair(ex, nk);
    *exec = ex; *n_kernels = nk;
    return LBM_OK;
}

// copy caller data (host or device) into a host vector
int to_host(const float *src, size_t count, std::vector<float> &dst)
{
    dst.resize(count);
    if (count == 0) return LBM_OK;
    if (is_device_ptr(src)) CK(cudaMemcpy(dst.data(), src, count * sizeof(float), cudaMemcpyDeviceToHost));
    else std::memcpy(dst.data(), src, count * sizeof(float));
    return LBM_OK;
}

// R17: the 4-cell stencil floor(x)-1 .. floor(x)+2 must stay inside 0..n-1 on wall axes
bool stencil_inside(const lbm *h, const double lo[3], const double hi[3])
{
    const int n[3] = {h->g.nx, h->g.ny, h->g.nz};
    const int wall[3] = {h->g.wallx, h->g.wally, h->g.wallz};
    for (int a = 0; a < 3; ++a) {
        if (!wall[a]) continue;
        if (std::floor(lo[a]) < 1.0 || std::floor(hi[a]) > (double)(n[a] - 3)) return false;
    }
    return true;
}

}  // namespace

// =================================================================================================
// Register the tiles n new markers occupy in their rest pose, for the tile edges 1, 2 and 4 (see auto_plan).
// Rotating bodies sweep other tiles later on, but about as many.
void count_rest_tiles(lbm *h, const float *pos, long long n)
{
    static const int edge[3] = {1, 2, 4};
    const Geom &g = h->g;
    for (int e = 0; e < 3; ++e) {
        const int tr = edge[e];
        const long long nty = (g.ny + tr - 1) / tr, ntz = (g.nz + tr - 1) / tr;
        const size_t slots = (size_t)(h->cg.nbx * nty * ntz);
        if (h->rest_map[e].size() != (slots + 63) / 64) { h->rest_map[e].assign((slots + 63) / 64, 0ull); h->rest_tiles[e] = 0; }
    }
    for (long long k = 0; k < n; ++k) {
        long long c[3];
        const int dim[3] = {g.nx, g.ny, g.nz};
        for (int a = 0; a < 3; ++a) {
            c[a] = (long long)std::floor((double)pos[3 * k + a]) % dim[a];
            if (c[a] < 0) c[a] += dim[a];
        }
        const long long blk = std::min<long long>(c[0] / CHUNK_W, h->cg.nbx - 1);
        for (int e = 0; e < 3; ++e) {
            const int tr = edge[e];
            const long long nty = (g.ny + tr - 1) / tr;
            const size_t slot = (size_t)(((c[2] / tr) * nty + c[1] / tr) * h->cg.nbx + blk);
            unsigned long long &w = h->rest_map[e][slot >> 6];
            const unsigned long long bit = 1ull << (slot & 63);
            if (!(w & bit)) { w |= bit; h->rest_tiles[e] += 1; }
        }
    }
}

extern "C" {

const char *lbm_last_error(void) { return g_err.c_str(); }

lbm_t *lbm_create(int nx, int ny, int nz, double tau, const lbm_bc_t *bc)
{
    if (nx < 1 || ny < 1 || nz < 1 || !(tau > 0.5) || !std::isfinite(tau)) {
        fail(LBM_EINVAL, "lbm_create: need nx,ny,nz >= 1 and tau > 0.5 (got %d %d %d %g)", nx, ny, nz, tau);
        return nullptr;
    }
    if ((long long)nx * ny * nz > 0x7fffffffLL / 2) {
        fail(LBM_EINVAL, "lbm_create: lattice too large for 32-bit cell keys");
        return nullptr;
    }
    lbm *h = new (std::nothrow) lbm();
    if (!h) { fail(LBM_ENOMEM, "lbm_create: host allocation failed"); return nullptr; }
    auto bail = [&](const char *what) -> lbm_t * {
        std::string msg = g_err;
        lbm_destroy(h);
        fail(LBM_ENOMEM, "lbm_create: %s: %s", what, msg.c_str());
        return nullptr;
    };
    if (cudaGetDevice(&h->device) != cudaSuccess) return bail("no CUDA device");
    h->g.nx = nx; h->g.ny = ny; h->g.nz = nz;
    h->g.nxw = (nx + 31) / 32;
    h->g.cells = (long long)nx * ny * nz;
    h->g.pitch = (h->g.cells + 3) / 4 * 4;   // plane padding was measured to make no difference (profiles/lbm_variants_r1.md)
    h->g.wallx = bc ? (bc->wall_x != 0) : 0;
    h->g.wally = bc ? (bc->wall_y != 0) : 0;
    h->g.wallz = bc ? (bc->wall_z != 0) : 0;
    h->tau = tau;
    h->cc.omega = (float)(1.0 / tau);
    h->cc.keep = (float)(1.0 - 1.0 / tau);
    h->cc.guo = (float)(1.0 - 0.5 / tau);
    h->cc.tau = (float)tau;
    h->cc.gbx = bc ? (float)bc->gx : 0.f;
    h->cc.gby = bc ? (float)bc->gy : 0.f;
    h->cc.gbz = bc ? (float)bc->gz : 0.f;
    h->cc.shift_forcing = 0;
    const size_t cells = (size_t)h->g.cells;
    h->n_mask_words = (size_t)h->g.nxw * ny * nz;
    {
        // capture streams: the MDF chain gets the highest priority, the bulk stream-collide the lowest, so the
        // short latency-bound IBM kernels are scheduled ahead of the lattice-wide pass they run beside
        int lo = 0, hi = 0;
        cudaDeviceGetStreamPriorityRange(&lo, &hi);
        bool ok = cudaStreamCreateWithPriority(&h->cap_stream, cudaStreamNonBlocking, hi) == cudaSuccess;
        ok &= cudaStreamCreateWithPriority(&h->cap_prep, cudaStreamNonBlocking, hi) == cudaSuccess;
        ok &= cudaStreamCreateWithPriority(&h->cap_prep2, cudaStreamNonBlocking, hi) == cudaSuccess;
        ok &= cudaStreamCreateWithPriority(&h->cap_bulk, cudaStreamNonBlocking, lo) == cudaSuccess;
        ok &= cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming) == cudaSuccess;
        ok &= cudaEventCreateWithFlags(&h->ev_bulk, cudaEventDisableTiming) == cudaSuccess;
        ok &= cudaEventCreateWithFlags(&h->ev_prep, cudaEventDisableTiming) == cudaSuccess;
        ok &= cudaEventCreateWithFlags(&h->ev_prep2, cudaEventDisableTiming) == cudaSuccess;
        ok &= cudaEventCreateWithFlags(&h->ev_mdf, cudaEventDisableTiming) == cudaSuccess;
        if (!ok) { fail(LBM_ECUDA, "%s", cudaGetErrorString(cudaGetLastError())); return bail("streams"); }
    }
    h->po = plane_offsets(h->g);
    const size_t fcount = (size_t)h->g.pitch * NQ;
    if (dmalloc(h, &h->f[0], fcount) || dmalloc(h, &h->f[1], fcount)) return bail("populations");
    if (dmalloc(h, &h->U, cells) || dmalloc(h, &h->G, cells)) return bail("U/G fields");
    if (dmalloc(h, &h->scal, (size_t)1)) return bail("scalars");
    h->cg = chunk_geom(nx);
    h->chunk_slots = (size_t)h->cg.nbx * ny * nz;
    h->tg = tile_geom(ny, nz);          // the tile tables are allocated with the markers (their edge depends on the set)
    bool ok = true;
    for (PrepSet &S : h->set) {
        if (dmalloc(h, &S.amask, h->n_mask_words) || dmalloc(h, &S.words, h->n_mask_words)) return bail("active mask");
        if (dmalloc(h, &S.chunk_of, h->chunk_slots)) return bail("chunk map");
        if (dmalloc(h, &S.scal, (size_t)1)) return bail("set scalars");
        // on a stream of the handle's own and with a stream synchronisation: a legacy-stream memset or a device-wide
        // synchronisation would collide with a graph capture another handle has open in another host thread
        ok &= cudaMemsetAsync(S.amask, 0, h->n_mask_words * sizeof(unsigned), h->cap_stream) == cudaSuccess;
        ok &= cudaMemsetAsync(S.chunk_of, 0xff, h->chunk_slots * sizeof(int), h->cap_stream) == cudaSuccess;
        ok &= cudaMemsetAsync(S.scal, 0, sizeof(SetScalars), h->cap_stream) == cudaSuccess;
    }
    ok &= cudaMemsetAsync(h->f[0], 0, fcount * sizeof(float), h->cap_stream) == cudaSuccess;   // rest state: f_i - t_i = 0
    ok &= cudaMemsetAsync(h->f[1], 0, fcount * sizeof(float), h->cap_stream) == cudaSuccess;
    ok &= cudaMemsetAsync(h->scal, 0, sizeof(DevScalars), h->cap_stream) == cudaSuccess;
    ok &= cudaStreamSynchronize(h->cap_stream) == cudaSuccess;
    if (!ok) { fail(LBM_ECUDA, "%s", cudaGetErrorString(cudaGetLastError())); return bail("memset"); }
    {
        int per_sm = 0, sms = 148;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, h->device);
        h->sms = sms;
        cudaFuncSetAttribute(k_spread_tiles, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)spread_tiles_smem(ChunkGeom{1, CHUNK_ENT_MAX}));
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_spread_tiles, TILE_WARPS * 32, spread_tiles_smem(h->cg));
        h->rows_grid = std::max(1, per_sm) * sms;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_stream_collide_words, 256, 0);
        h->words_grid = std::max(1, per_sm) * sms;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_moments_active, 256, 0);
        h->moments_grid = std::max(1, per_sm) * sms;
    }
    g_err.clear();
    return h;
}

void lbm_destroy(lbm_t *h)
{
    if (!h) return;
    // wait for the handle's own work only (never the whole device: a device-wide synchronisation fails while another
    // handle captures a graph in another host thread, and invalidates that capture)
    cudaStreamSynchronize(h->stream);
    if (h->copy_stream) cudaStreamSynchronize(h->copy_stream);
    drop_graphs(h);
    free_markers_dev(h);
    cudaFree(h->f[0]); cudaFree(h->f[1]); cudaFree(h->U); cudaFree(h->G); cudaFree(h->scal);
    for (PrepSet &S : h->set) {
        cudaFree(S.amask); cudaFree(S.words); cudaFree(S.chunk_of); cudaFree(S.bin_first); cudaFree(S.scal);
    }
    for (int a = 0; a < 3; ++a) cudaFree(h->stage[a]);
    cudaFree(h->async_stage);
    if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
    if (h->ev_pack) cudaEventDestroy(h->ev_pack);
    if (h->ev_copy) cudaEventDestroy(h->ev_copy);
    if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
    if (h->cap_bulk) cudaStreamDestroy(h->cap_bulk);
    if (h->cap_prep) cudaStreamDestroy(h->cap_prep);
    if (h->cap_prep2) cudaStreamDestroy(h->cap_prep2);
    if (h->ev_fork) cudaEventDestroy(h->ev_fork);
    if (h->ev_bulk) cudaEventDestroy(h->ev_bulk);
    if (h->ev_prep) cudaEventDestroy(h->ev_prep);
    if (h->ev_prep2) cudaEventDestroy(h->ev_prep2);
    if (h->ev_mdf) cudaEventDestroy(h->ev_mdf);
    drop_traces(h);
    delete h;
}

const char *lbm_trace_label(lbm_t *h, int i)
{
    if (!h || !h->trace_last || i < 0 || (size_t)i >= h->trace_last->label.size()) return "";
    return h->trace_last->label[(size_t)i].c_str();
}

int lbm_query_layout(int nx, int ny, int nz, int *out)
{
    if (nx < 1 || ny < 1 || nz < 1 || !out) return fail(LBM_EINVAL, "lbm_query_layout: bad arguments");
    const ChunkGeom cg = chunk_geom(nx);
    const TileGeom tg = tile_geom(ny, nz);   // for the 4 x 4-row tiles of large marker sets
    out[0] = cg.nbx; out[1] = cg.ent; out[2] = tg.nty; out[3] = tg.ntz; out[4] = (nx + 31) / 32;
    out[5] = CHUNK_W; out[6] = TILE_R; out[7] = CHUNK_ENT_MAX;
    return LBM_OK;
}

int lbm_set_stream(lbm_t *h, void *cuda_stream)
{
    if (!h) return fail(LBM_EINVAL, "lbm_set_stream: NULL handle");
    if (h->stream != (cudaStream_t)cuda_stream) CK(cudaStreamSynchronize(h->stream));
    h->stream = (cudaStream_t)cuda_stream;
    return LBM_OK;
}

int lbm_set_option(lbm_t *h, int key, int value)
{
    if (!h) return fail(LBM_EINVAL, "lbm_set_option: NULL handle");
    switch (key) {
        case LBM_OPT_SPREAD: if (value < 0 || value > 3) break; h->opt_spread = value; return LBM_OK;
        case LBM_OPT_FORCING: if (value < 0 || value > 1) break; h->opt_forcing = value; return LBM_OK;
        case LBM_OPT_GRAPH: if (value < 0 || value > 1) break; h->opt_graph = value; return LBM_OK;
        case LBM_OPT_LBM_KERNEL: if (value < 0 || value > 2) break; h->opt_lbm_kernel = value; return LBM_OK;
        case LBM_OPT_OVERLAP: if (value < 0 || value > 3) break; h->opt_overlap = value; return LBM_OK;
        case LBM_OPT_MOMENTS: if (value < 0 || value > 2) break; h->opt_moments = value; return LBM_OK;
        case LBM_OPT_INTERP: if (value < 0 || value > 3) break; h->opt_interp = value; return LBM_OK;
        case LBM_OPT_TIMING: if (value < 0 || value > 1) break; h->opt_timing = value; h->timer.reset(); return LBM_OK;
        case LBM_OPT_FUSED: if (value < 0 || value > 1) break; h->opt_fused = value; return LBM_OK;
        case LBM_OPT_TILE_ROWS: if (value != 0 && value != 1 && value != 2 && value != 4) break; h->opt_tile_rows = value; return LBM_OK;
        case LBM_OPT_PERSISTENT: if (value < 0 || value > 2) break; h->opt_persistent = value; return LBM_OK;
        case LBM_OPT_MDF_BLOCKS:
            if (value < 0 || value > 32) break;
            h->opt_mdf_blocks = value;
            if (h->tr > 0) {                       // cached graphs hold the old grids
                CK(cudaStreamSynchronize(h->stream));
                drop_graphs(h);
                int rc = mdf_launch_geometry(h);
                if (rc) return rc;
            }
            return LBM_OK;
        case LBM_OPT_TILE_WARPS: if (value < 0 || value > 2) break; h->opt_tile_warps = value; return LBM_OK;
        case LBM_OPT_PIPELINE: if (value < 0 || value > 2) break; h->opt_pipeline = value; return LBM_OK;
        case LBM_OPT_BULK_STREAM: if (value < 0 || value > 2) break; h->opt_bulk_stream = value; return LBM_OK;
        case LBM_OPT_TRACE:
            if (value < 0 || value > 1) break;
            if (value != h->opt_trace) { CK(cudaStreamSynchronize(h->stream)); drop_graphs(h); h->opt_trace = value; }
            return LBM_OK;
        case LBM_OPT_TILE_CAP:
            if (value < 0) break;
            if (value != h->opt_tile_cap) { h->opt_tile_cap = value; h->realloc_tables = true; h->markers_stale = true; }
            return LBM_OK;
        default: return fail(LBM_EINVAL, "lbm_set_option: unknown key %d", key);
    }
    return fail(LBM_EINVAL, "lbm_set_option: value %d out of range for key %d", value, key);
}

int lbm_get_info(lbm_t *h, int key, long long *value)
{
    if (!h || !value) return fail(LBM_EINVAL, "lbm_get_info: NULL argument");
    switch (key) {
        case LBM_INFO_MARKERS: *value = (long long)h->h_area.size(); return LBM_OK;
        case LBM_INFO_BODIES: *value = (long long)h->bodies.size(); return LBM_OK;
        case LBM_INFO_STEPS: *value = h->steps_done; return LBM_OK;
        case LBM_INFO_LAUNCHES: *value = h->launches; return LBM_OK;
        case LBM_INFO_DEVICE_BYTES: *value = (long long)h->dev_bytes; return LBM_OK;
        case LBM_INFO_ACTIVE_CELLS: case LBM_INFO_RUNS: case LBM_INFO_RUN_ENTRIES: case LBM_INFO_TILES:
        case LBM_INFO_ACTIVE_WORDS: {
            int r = 0;
            if (h->force_valid && h->last_set >= 0) {
                const SetScalars *sc = h->set[h->last_set].scal;
                const int *p = key == LBM_INFO_ACTIVE_CELLS ? &sc->n_cells : (key == LBM_INFO_RUNS ? &sc->n_chunks : (key == LBM_INFO_TILES ? &sc->n_tiles : (key == LBM_INFO_ACTIVE_WORDS ? &sc->n_words : &sc->n_entries)));
                CK(cudaMemcpyAsync(&r, p, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
                CK(cudaStreamSynchronize(h->stream));
            }
            *value = r;
            return LBM_OK;
        }
        case LBM_INFO_STATUS: {
            int st = 0;
            CK(cudaMemcpyAsync(&st, &h->scal->status, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
            CK(cudaStreamSynchronize(h->stream));
            *value = st;
            return LBM_OK;
        }
        case LBM_INFO_TRACE_COUNT: *value = h->trace_last ? (long long)h->trace_last->ev.size() : 0; return LBM_OK;
        case LBM_INFO_LAYOUT: *value = (h->nm > 0) ? overlap_mode(h) : 0; return LBM_OK;
        case LBM_INFO_TILE_ROWS: *value = h->tr; return LBM_OK;
        case LBM_INFO_SORT_PASSES: *value = h->sort_passes; return LBM_OK;
        default:
            if (h->trace_last && key >= LBM_INFO_TRACE_NS && key < LBM_INFO_TRACE_NS + (int)h->trace_last->ev.size()) {
                // device time from the first trace event of the last step (the fork) to event key - LBM_INFO_TRACE_NS
                CK(cudaStreamSynchronize(h->stream));
                float ms = 0.f;
                CK(cudaEventElapsedTime(&ms, h->trace_last->ev[0], h->trace_last->ev[(size_t)(key - LBM_INFO_TRACE_NS)]));
                *value = (long long)(1e6 * (double)ms);
                return LBM_OK;
            }
            if (key >= LBM_INFO_PHASE_NS && key < LBM_INFO_PHASE_NS + PH_COUNT) {
                *value = (long long)h->timer.ns[key - LBM_INFO_PHASE_NS];
                return LBM_OK;
            }
            return fail(LBM_EINVAL, "lbm_get_info: unknown key %d", key);
    }
}

int lbm_set_fields(lbm_t *h, const float *rho, const float *u)
{
    if (!h) return fail(LBM_EINVAL, "lbm_set_fields: NULL handle");
    int rc = flush_ibm(h);
    if (rc) return rc;
    const size_t cells = (size_t)h->g.cells;
    const float *p_rho = rho, *p_u = u;
    // host sources go through the handle's staging buffers (kept between calls: no cudaMalloc / cudaFree, which
    // synchronise the device, on the path of a host loop that resets the fields)
    if (rho && !is_device_ptr(rho)) {
        float *d = (float *)stage_get(h, 0, cells * sizeof(float));
        if (!d) return fail(LBM_ENOMEM, "lbm_set_fields: staging allocation failed");
        CK(cudaMemcpyAsync(d, rho, cells * sizeof(float), cudaMemcpyHostToDevice, h->stream));
        p_rho = d;
    }
    if (u && !is_device_ptr(u)) {
        float *d = (float *)stage_get(h, 1, 3 * cells * sizeof(float));
        if (!d) return fail(LBM_ENOMEM, "lbm_set_fields: staging allocation failed");
        CK(cudaMemcpyAsync(d, u, 3 * cells * sizeof(float), cudaMemcpyHostToDevice, h->stream));
        p_u = d;
    }
    dim3 b = cell_block(h->g);
    k_init_fields<<<cell_grid(h->g, b), b, 0, h->stream>>>(h->f[h->cur], h->g, p_rho, p_u);
    h->launches += 1;
    cudaError_t e = cudaGetLastError();
    // the caller's host buffers may be reused when the call returns
    if (e == cudaSuccess && (p_rho != rho || p_u != u)) e = cudaStreamSynchronize(h->stream);
    stage_release(h);
    if (e != cudaSuccess) return fail(LBM_ECUDA, "lbm_set_fields: %s", cudaGetErrorString(e));
    h->steps_done = 0;
    h->force_valid = false;
    return LBM_OK;
}

int ibm_set_markers(lbm_t *h, const float *pos, const float *vel, const float *area, long long n)
{
    if (!h) return fail(LBM_EINVAL, "ibm_set_markers: NULL handle");
    if (n < 0 || (n > 0 && (!pos || !area))) return fail(LBM_EINVAL, "ibm_set_markers: bad arguments");
    if ((long long)h->h_area.size() + n > 0x7fffffffLL / 4) return fail(LBM_EINVAL, "ibm_set_markers: too many markers");
    if (n > 0 && (h->g.nx < 4 || h->g.ny < 4 || h->g.nz < 4))
        return fail(LBM_EINVAL, "ibm_set_markers: the lattice must be at least 4 cells wide on every axis");
    std::vector<float> p, v, s;
    int rc;
    if ((rc = to_host(pos, (size_t)(3 * n), p))) return rc;
    if ((rc = to_host(area, (size_t)n, s))) return rc;
    if (vel) { if ((rc = to_host(vel, (size_t)(3 * n), v))) return rc; }
    else v.assign((size_t)(3 * n), 0.f);
    // static body until ibm_set_kinematics: centre := centroid (only used to keep fp32 offsets small)
    HostBody B{};
    B.first = (long long)h->h_area.size(); B.count = n; B.omega = 0.0;
    B.axis[0] = 0.0; B.axis[1] = 0.0; B.axis[2] = 1.0; B.has_kin = false;
    double c[3] = {0, 0, 0};
    for (long long k = 0; k < n; ++k) {
        double x[3] = {p[(size_t)(3 * k)], p[(size_t)(3 * k + 1)], p[(size_t)(3 * k + 2)]};
        if (!std::isfinite(x[0]) || !std::isfinite(x[1]) || !std::isfinite(x[2]) || !std::isfinite(s[(size_t)k]) ||
            !std::isfinite(v[(size_t)(3 * k)]) || !std::isfinite(v[(size_t)(3 * k + 1)]) || !std::isfinite(v[(size_t)(3 * k + 2)]))
            return fail(LBM_EINVAL, "ibm_set_markers: non-finite input at marker %lld", k);
        if (!stencil_inside(h, x, x))
            return fail(LBM_ERANGE, "ibm_set_markers: stencil of marker %lld (%.3f %.3f %.3f) crosses a wall", k,
                        x[0], x[1], x[2]);
        for (int a = 0; a < 3; ++a) c[a] += x[a];
    }
    for (int a = 0; a < 3; ++a) B.center[a] = n > 0 ? c[a] / (double)n : 0.0;
    count_rest_tiles(h, p.data(), n);
    h->h_pos.insert(h->h_pos.end(), p.begin(), p.end());
    h->h_vel.insert(h->h_vel.end(), v.begin(), v.end());
    h->h_area.insert(h->h_area.end(), s.begin(), s.end());
    h->h_body.insert(h->h_body.end(), (size_t)n, (int)h->bodies.size());
    h->bodies.push_back(B);
    h->markers_stale = true;
    return (int)h->bodies.size() - 1;
}

int ibm_set_kinematics(lbm_t *h, double omega, const double *axis, const double *center)
{
    if (!h || !axis || !center) return fail(LBM_EINVAL, "ibm_set_kinematics: NULL argument");
    if (h->bodies.empty()) return fail(LBM_ESTATE, "ibm_set_kinematics: no body defined yet");
    const double nrm = std::sqrt(axis[0] * axis[0] + axis[1] * axis[1] + axis[2] * axis[2]);
    if (!(nrm > 0.0) || !std::isfinite(nrm) || !std::isfinite(omega))
        return fail(LBM_EINVAL, "ibm_set_kinematics: axis must be non-zero and finite");
    if (!std::isfinite(center[0]) || !std::isfinite(center[1]) || !std::isfinite(center[2]))
        return fail(LBM_EINVAL, "ibm_set_kinematics: non-finite centre");
    HostBody &B = h->bodies.back();
    if (omega != 0.0) {
        // every point stays on a sphere of radius |p - c| about c
        for (long long k = B.first; k < B.first + B.count; ++k) {
            double r2 = 0.0;
            for (int a = 0; a < 3; ++a) {
                const double d = (double)h->h_pos[(size_t)(3 * k + a)] - center[a];
                r2 += d * d;
            }
            const double r = std::sqrt(r2);
            const double lo[3] = {center[0] - r, center[1] - r, center[2] - r};
            const double hi[3] = {center[0] + r, center[1] + r, center[2] + r};
            if (!stencil_inside(h, lo, hi))
                return fail(LBM_ERANGE, "ibm_set_kinematics: marker %lld (radius %.3f) can reach a wall", k, r);
        }
    }
    B.omega = omega;
    for (int a = 0; a < 3; ++a) { B.axis[a] = axis[a] / nrm; B.center[a] = center[a]; }
    B.has_kin = true;
    h->markers_stale = true;
    return LBM_OK;
}

int ibm_update_kinematics(lbm_t *h, int first_body, int count, const double *omega, const double *axis,
                          const double *center)
{
    if (!h || !omega || !axis) return fail(LBM_EINVAL, "ibm_update_kinematics: NULL argument");
    if (first_body < 0 || count < 0 || (size_t)first_body + (size_t)count > h->bodies.size())
        return fail(LBM_EINVAL, "ibm_update_kinematics: body range out of bounds");
    std::vector<HostBody> nb(h->bodies.begin() + first_body, h->bodies.begin() + first_body + count);
    bool moved = false;
    for (int b = 0; b < count; ++b) {
        const double *ax = axis + 3 * b;
        const double nrm = std::sqrt(ax[0] * ax[0] + ax[1] * ax[1] + ax[2] * ax[2]);
        if (!(nrm > 0.0) || !std::isfinite(nrm) || !std::isfinite(omega[b]))
            return fail(LBM_EINVAL, "ibm_update_kinematics: bad axis or omega for body %d", first_body + b);
        HostBody &B = nb[(size_t)b];
        const double *c = center ? center + 3 * b : B.center;
        if (!std::isfinite(c[0]) || !std::isfinite(c[1]) || !std::isfinite(c[2]))
            return fail(LBM_EINVAL, "ibm_update_kinematics: non-finite centre for body %d", first_body + b);
        if (center) for (int a = 0; a < 3; ++a) moved |= (c[a] != B.center[a]);
        const bool any_wall = h->g.wallx || h->g.wally || h->g.wallz;
        if (any_wall && omega[b] != 0.0 && (center || B.omega == 0.0))
            for (long long k = B.first; k < B.first + B.count; ++k) {
                double r2 = 0.0;
                for (int a = 0; a < 3; ++a) {
                    const double d = (double)h->h_pos[(size_t)(3 * k + a)] - c[a];
                    r2 += d * d;
                }
                const double r = std::sqrt(r2);
                const double lo[3] = {c[0] - r, c[1] - r, c[2] - r}, hi[3] = {c[0] + r, c[1] + r, c[2] + r};
                if (!stencil_inside(h, lo, hi))
                    return fail(LBM_ERANGE, "ibm_update_kinematics: marker %lld can reach a wall", k);
            }
        B.omega = omega[b];
        for (int a = 0; a < 3; ++a) { B.axis[a] = ax[a] / nrm; B.center[a] = c[a]; }
        B.has_kin = true;
    }
    bool changed = moved;
    for (int b = 0; b < count && !changed; ++b) {
        const HostBody &o = h->bodies[(size_t)(first_body + b)], &n = nb[(size_t)b];
        changed = o.omega != n.omega || o.axis[0] != n.axis[0] || o.axis[1] != n.axis[1] || o.axis[2] != n.axis[2];
    }
    std::copy(nb.begin(), nb.end(), h->bodies.begin() + first_body);
    if (moved || h->markers_stale) { h->markers_stale = true; return LBM_OK; }
    // a set prepared ahead for the next step used the old table
    if (changed) for (PrepSet &S : h->set) if (S.step >= h->steps_done) { S.step = -1; S.stage = 0; }
    // centres unchanged: only the small per-body table changes; graphs and marker arrays stay valid
    for (int b = 0; b < count; ++b) {
        const HostBody &B = h->bodies[(size_t)(first_body + b)];
        BodyDef &d = h->h_defs[(size_t)(first_body + b)];
        d.omega = B.omega; d.ax = B.axis[0]; d.ay = B.axis[1]; d.az = B.axis[2];
    }
    CK(cudaMemcpyAsync(h->d_defs + first_body, h->h_defs.data() + first_body, sizeof(BodyDef) * (size_t)count,
                       cudaMemcpyHostToDevice, h->stream));
    return LBM_OK;
}

int ibm_clear(lbm_t *h)
{
    if (!h) return fail(LBM_EINVAL, "ibm_clear: NULL handle");
    int rc = flush_ibm(h);
    if (rc) return rc;
    h->h_pos.clear(); h->h_vel.clear(); h->h_area.clear(); h->h_body.clear(); h->bodies.clear();
    for (int e = 0; e < 3; ++e) { h->rest_map[e].clear(); h->rest_tiles[e] = 0; }
    h->markers_stale = true;
    return LBM_OK;
}

int lbm_ibm_step(lbm_t *h, int nsteps, int mdf_iters)
{
    if (!h) return fail(LBM_EINVAL, "lbm_ibm_step: NULL handle");
    if (nsteps < 0 || mdf_iters < 0) return fail(LBM_EINVAL, "lbm_ibm_step: negative count");
    if (mdf_iters > MAX_MDF) return fail(LBM_EINVAL, "lbm_ibm_step: at most %d MDF iterations", MAX_MDF);
    if (nsteps == 0) return LBM_OK;
    if (effective_tr(h) != h->tr) h->markers_stale = true;      // an option changed the tile edge: rebuild the tables
    int rc = upload_markers(h);
    if (rc) return rc;
    const bool ibm = (h->nm > 0 && mdf_iters > 0);
    if (!ibm) { if ((rc = flush_ibm(h))) return rc; }
    if (ibm) {
        k_set_scalars<<<1, 1, 0, h->stream>>>(&h->scal->step_ctr, h->steps_done, nullptr, 0, 1);
        h->launches += 1;
        if (h->opt_spread != 0)
            for (PrepSet &S : h->set) if ((rc = ensure_bin_first(h, S))) return rc;
        if ((rc = ensure_comparison_arrays(h))) return rc;
    }
    const bool overlapped = ibm && h->opt_overlap && h->opt_graph && !h->opt_timing;
    if (overlapped) {
        // the steady-state graphs of every (buffer parity, marker set) combination are built now, not one by one
        // during the first six steps of a run
        const int pipe = pipeline_depth(h) == 2 ? 3 : 0;
        for (int par = 0; par < 2; ++par)
            for (int st = 0; st < N_SETS; ++st) {
                cudaGraphExec_t ex = nullptr;
                int nk = 0;
                if ((rc = get_graph(h, 2, par, st, mdf_iters, &ex, &nk, pipe))) return rc;
            }
    }
    for (int s = 0; s < nsteps; ++s) {
        int nk = 0;
        cudaGraphExec_t ex = nullptr;
        PrepSet *S = ibm ? &h->set[h->cur_set] : nullptr;
        if (overlapped) {
            const int sig = prep_signature(h);
            const int depth2 = pipeline_depth(h) == 2;
            if (S->step != h->steps_done || S->spread != sig || S->stage != 2) {
                // first step of a run (or the kinematics changed): bin this step's markers in line -- all of it, or the
                // second half if the set already holds this step's sorted keys
                const bool half = S->step == h->steps_done && S->spread == sig && S->stage == 1;
                int np = 0;
                if ((rc = enqueue_prep(h, h->stream, *S, 0, &np, nullptr, half ? PREP_BINS : PREP_ALL))) return rc;
                h->launches += np;
                S->step = h->steps_done; S->spread = sig; S->stage = 2; S->dirty = true;
            }
            PrepSet &N = h->set[(h->cur_set + 1) % N_SETS];
            const bool n_has_sort = N.step == h->steps_done + 1 && N.spread == sig && N.stage == 1;
            if ((rc = get_graph(h, 2, h->cur, h->cur_set, mdf_iters, &ex, &nk, (n_has_sort ? 1 : 0) | (depth2 ? 2 : 0)))) return rc;
            CK(cudaGraphLaunch(ex, h->stream));
            if (h->opt_trace) { auto tr = h->traces.find(h->last_key); h->trace_last = tr == h->traces.end() ? nullptr : &tr->second; }
            N.step = h->steps_done + 1; N.spread = sig; N.stage = 2; N.dirty = true;
            if (depth2) {
                PrepSet &N2 = h->set[(h->cur_set + 2) % N_SETS];
                N2.step = h->steps_done + 2; N2.spread = sig; N2.stage = 1; N2.dirty = true;
            }
            h->last_set = h->cur_set;
            h->cur_set = (h->cur_set + 1) % N_SETS;
        } else {
            if (h->opt_timing) {
                if ((rc = enqueue_step_serial(h, h->stream, h->cur, S, true, mdf_iters, &nk, &h->timer))) return rc;
                CK(cudaStreamSynchronize(h->stream));
                h->timer.collect();
            } else if (h->opt_graph) {
                if ((rc = get_graph(h, ibm ? 1 : 0, h->cur, h->cur_set, mdf_iters, &ex, &nk))) return rc;
                CK(cudaGraphLaunch(ex, h->stream));
            } else {
                if ((rc = enqueue_step_serial(h, h->stream, h->cur, S, true, mdf_iters, &nk))) return rc;
            }
            if (S) { S->step = h->steps_done; S->spread = prep_signature(h); S->stage = 2; S->dirty = true; h->last_set = h->cur_set; }
        }
        h->launches += nk;
        h->cur ^= 1;
        h->steps_done += 1;
        if (ibm) h->force_valid = true;
    }
    return LBM_OK;
}

int lbm_read_fields(lbm_t *h, float *rho, float *u, float *force)
{
    if (!h) return fail(LBM_EINVAL, "lbm_read_fields: NULL handle");
    if (!rho && !u && !force) return LBM_OK;
    const size_t cells = (size_t)h->g.cells;
    float *out[3] = {rho, u, force};
    const size_t cnt[3] = {cells, 3 * cells, 3 * cells};
    float *dev[3] = {nullptr, nullptr, nullptr};
    bool tmp[3] = {false, false, false};
    for (int a = 0; a < 3; ++a) {
        if (!out[a]) continue;
        if (is_device_ptr(out[a])) dev[a] = out[a];
        else {
            if (!(dev[a] = (float *)stage_get(h, a, cnt[a] * sizeof(float)))) {
                stage_release(h);
                return fail(LBM_ENOMEM, "lbm_read_fields: staging allocation failed");
            }
            tmp[a] = true;
        }
    }
    dim3 b = cell_block(h->g);
    const unsigned *mask = (h->force_valid && h->last_set >= 0) ? h->set[h->last_set].amask : nullptr;
    k_read_fields<<<cell_grid(h->g, b), b, 0, h->stream>>>(h->f[h->cur], h->g, mask, h->G, dev[0], dev[1], dev[2]);
    h->launches += 1;
    cudaError_t e = cudaGetLastError();
    bool any_tmp = false;
    for (int a = 0; a < 3 && e == cudaSuccess; ++a)
        if (tmp[a]) {
            any_tmp = true;
            e = cudaMemcpyAsync(out[a], dev[a], cnt[a] * sizeof(float), cudaMemcpyDeviceToHost, h->stream);
        }
    if (any_tmp && e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    stage_release(h);
    if (e != cudaSuccess) return fail(LBM_ECUDA, "lbm_read_fields: %s", cudaGetErrorString(e));
    return LBM_OK;
}

int ibm_read_markers(lbm_t *h, float *pos, float *force, int *perm, int *cell)
{
    if (!h) return fail(LBM_EINVAL, "ibm_read_markers: NULL handle");
    const int n = (int)h->h_area.size();
    if (n == 0 || (!pos && !force && !perm && !cell)) return LBM_OK;
    if (h->last_set < 0 || h->markers_stale)
        return fail(LBM_ESTATE, "ibm_read_markers: no IBM step has been run with the current markers");
    const PrepSet &S = h->set[h->last_set];
    const unsigned *skey = sorted_keys(h, S);
    const int *dperm = sorted_perm(h, S);
    void *out[3] = {pos, force, cell};
    const size_t bytes[3] = {sizeof(float) * 3 * (size_t)n, sizeof(float) * 3 * (size_t)n, sizeof(int) * (size_t)n};
    void *dev[3] = {nullptr, nullptr, nullptr};
    bool tmp[3] = {false, false, false};
    for (int a = 0; a < 3; ++a) {
        if (!out[a]) continue;
        if (is_device_ptr(out[a])) dev[a] = out[a];
        else {
            if (!(dev[a] = stage_get(h, a, bytes[a]))) return fail(LBM_ENOMEM, "ibm_read_markers: staging allocation failed");
            tmp[a] = true;
        }
    }
    k_read_markers<<<(n + 255) / 256, 256, 0, h->stream>>>(skey, dperm, n, h->g, S.ms.fs, S.ms.du, (float *)dev[0],
                                                            (float *)dev[1], (int *)dev[2]);
    h->launches += 1;
    cudaError_t e = cudaGetLastError();
    bool need_sync = false;
    for (int a = 0; a < 3 && e == cudaSuccess; ++a)
        if (tmp[a]) { need_sync = true; e = cudaMemcpyAsync(out[a], dev[a], bytes[a], cudaMemcpyDeviceToHost, h->stream); }
    if (perm && e == cudaSuccess) {
        const bool dv = is_device_ptr(perm);
        e = cudaMemcpyAsync(perm, dperm, sizeof(int) * (size_t)n, dv ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost,
                            h->stream);
        need_sync |= !dv;
    }
    if (need_sync && e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    stage_release(h);
    if (e != cudaSuccess) return fail(LBM_ECUDA, "ibm_read_markers: %s", cudaGetErrorString(e));
    return LBM_OK;
}

int ibm_read_markers_async(lbm_t *h, float *force)
{
    if (!h || !force) return fail(LBM_EINVAL, "ibm_read_markers_async: NULL argument");
    const int n = (int)h->h_area.size();
    if (n == 0) return LBM_OK;
    if (h->last_set < 0 || h->markers_stale)
        return fail(LBM_ESTATE, "ibm_read_markers_async: no IBM step has been run with the current markers");
    if (!h->copy_stream) {
        CK(cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
        CK(cudaEventCreateWithFlags(&h->ev_pack, cudaEventDisableTiming));
        CK(cudaEventCreateWithFlags(&h->ev_copy, cudaEventDisableTiming));
    }
    const size_t bytes = sizeof(float) * 3 * (size_t)n;
    if (h->async_cap < bytes) {
        if (h->copy_pending) CK(cudaEventSynchronize(h->ev_copy));
        if (h->async_stage) { cudaFree(h->async_stage); h->dev_bytes -= h->async_cap; h->async_stage = nullptr; h->async_cap = 0; }
        CK(cudaMalloc((void **)&h->async_stage, bytes));
        h->async_cap = bytes; h->dev_bytes += bytes;
    }
    // the packing kernel must not overwrite the staging buffer while the previous copy still reads it
    if (h->copy_pending) CK(cudaStreamWaitEvent(h->stream, h->ev_copy, 0));
    const PrepSet &S = h->set[h->last_set];
    k_read_markers<<<(n + 255) / 256, 256, 0, h->stream>>>(sorted_keys(h, S), sorted_perm(h, S), n, h->g, S.ms.fs, S.ms.du,
                                                            nullptr, h->async_stage, nullptr);
    h->launches += 1;
    CK(cudaGetLastError());
    CK(cudaEventRecord(h->ev_pack, h->stream));
    CK(cudaStreamWaitEvent(h->copy_stream, h->ev_pack, 0));
    CK(cudaMemcpyAsync(force, h->async_stage, bytes, cudaMemcpyDeviceToHost, h->copy_stream));
    CK(cudaEventRecord(h->ev_copy, h->copy_stream));
    h->copy_pending = true;
    return LBM_OK;
}

int ibm_wait_markers(lbm_t *h)
{
    if (!h) return fail(LBM_EINVAL, "ibm_wait_markers: NULL handle");
    if (h->copy_pending) { CK(cudaEventSynchronize(h->ev_copy)); h->copy_pending = false; }
    return LBM_OK;
}

int lbm_sync(lbm_t *h)
{
    if (!h) return fail(LBM_EINVAL, "lbm_sync: NULL handle");
    int st = 0;
    CK(cudaMemcpyAsync(&st, &h->scal->status, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    if (h->copy_pending) { CK(cudaEventSynchronize(h->ev_copy)); h->copy_pending = false; }
    if (st) {
        CK(cudaMemsetAsync(&h->scal->status, 0, sizeof(int), h->stream));
        if (st & 2)
            return fail(LBM_ENOMEM, "lbm_sync: more marker chunks / tiles than the tables hold (%d / %d) during the last steps",
                        h->chunk_cap, h->tile_cap);
        return fail(LBM_ERANGE, "lbm_sync: a marker stencil crossed a wall face during the last steps");
    }
    return LBM_OK;
}

}  // extern "C"

// ---- a3 without any allocation: ibm_sort_cells_noalloc -------------------------------------------------------------
// The stable LSD radix sort of the binning (sort_kernels.cuh: k_radix_hist / k_radix_scan / k_radix_scatter, the very
// kernels the step uses above 32,768 markers) for callers that cannot call cudaMalloc (code under CUDA graph capture,
// tight serving loops, harnesses that forbid it).  The scratch the sort needs -- the per-sub-tile digit histograms, the
// digit totals and one ping-pong copy of keys and values -- lives in a file-scope device array of fixed size; every GPU
// that loads the library holds these 3 MiB + 1 KiB until the process exits.
//
// g_noalloc_scratch below is, in HOST code, only a stand-in for the symbol: its address is NOT a device address.  The
// device address comes from cudaGetSymbolAddress, asked for once per device with that device current
// (noalloc_scratch_ptr), and that pointer is what the kernels are given.
namespace {

constexpr int NOALLOC_MAX_MARKERS = 262144;      // stated maximum of ibm_sort_cells_noalloc (IBM_NOALLOC_MAX_MARKERS)
constexpr int NOALLOC_MAX_TILES = 1024;          // sub-tiles of the sort (one warp each) at the maximum
struct NoallocScratch {
    unsigned keys[NOALLOC_MAX_MARKERS];          // ping-pong partner of the caller's key output
    int vals[NOALLOC_MAX_MARKERS];               // ping-pong partner of the caller's permutation output
    int hist[RADIX * NOALLOC_MAX_TILES];         // [digit][sub-tile], fully rewritten by every pass
    int total[RADIX];                            // digit totals, fully rewritten by every pass
};
static_assert(NOALLOC_MAX_MARKERS == IBM_NOALLOC_MAX_MARKERS, "lbm_ibm.h states the maximum");
static_assert(sizeof(NoallocScratch) == 3 * 1048576 + 1024, "the header and README state 3 MiB + 1 KiB");

}  // namespace

static __device__ __align__(256) unsigned char g_noalloc_scratch[sizeof(NoallocScratch)];

namespace {

constexpr int NOALLOC_MAX_DEVICES = 64;
NoallocScratch *g_noalloc_ptr[NOALLOC_MAX_DEVICES];       // device address of g_noalloc_scratch on device i, or NULL
std::mutex g_noalloc_mutex;

// Device address of the scratch array on the CURRENT device (asked for once per device).  No allocation: the array
// is part of the loaded module.
int noalloc_scratch_ptr(NoallocScratch **out)
{
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(LBM_EINVAL, "ibm_sort_cells_noalloc: device ordinal %d not supported", dev);
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
        void *p = nullptr;
        CK(cudaGetSymbolAddress(&p, g_noalloc_scratch));
        if (!p) return fail(LBM_ECUDA, "ibm_sort_cells_noalloc: cudaGetSymbolAddress returned a NULL address");
        g_noalloc_ptr[dev] = static_cast<NoallocScratch *>(p);
    }
    *out = g_noalloc_ptr[dev];
    return LBM_OK;
}

}  // namespace

extern "C" int ibm_sort_cells_noalloc(const unsigned *cell, int n, long long ncells, unsigned *cell_sorted, int *perm,
                                      void *cuda_stream)
{
    if (n < 0) return fail(LBM_EINVAL, "ibm_sort_cells_noalloc: n = %d < 0", n);
    if (n > NOALLOC_MAX_MARKERS)
        return fail(LBM_ERANGE, "ibm_sort_cells_noalloc: n = %d exceeds the fixed scratch array (at most %d markers); "
                                "use the handle-based path (ibm_set_markers + lbm_ibm_step) for larger sets",
                    n, NOALLOC_MAX_MARKERS);
    if (ncells < 1 || ncells > (1ll << 32)) return fail(LBM_EINVAL, "ibm_sort_cells_noalloc: ncells = %lld out of range", ncells);
    if (n == 0) return LBM_OK;
    if (!cell || !cell_sorted || !perm) return fail(LBM_EINVAL, "ibm_sort_cells_noalloc: NULL buffer");
    if (!is_device_ptr(cell) || !is_device_ptr(cell_sorted) || !is_device_ptr(perm))
        return fail(LBM_EINVAL, "ibm_sort_cells_noalloc: cell, cell_sorted and perm must be device pointers");
    if ((const void *)cell == (const void *)cell_sorted) return fail(LBM_EINVAL, "ibm_sort_cells_noalloc: cell_sorted must not alias cell");
    NoallocScratch *sc = nullptr;
    int rc = noalloc_scratch_ptr(&sc);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    // sort geometry: as in the handle-based path, with sub-tiles widened until they fit the fixed histogram table
    // (the result of a stable sort does not depend on it)
    int ipw = ((n / (148 * 32)) + 31) / 32 * 32;
    ipw = std::max(ipw, ((n + NOALLOC_MAX_TILES - 1) / NOALLOC_MAX_TILES + 31) / 32 * 32);
    ipw = std::min(std::max(ipw, 64), 2048);
    const int tiles = (n + ipw - 1) / ipw;
    if (tiles > NOALLOC_MAX_TILES) return fail(LBM_ERANGE, "ibm_sort_cells_noalloc: %d sub-tiles exceed the scratch array", tiles);
    int bits = 1;
    while (bits < 32 && (1ll << bits) < ncells) ++bits;
    const int passes = (bits + 7) / 8;
    const int sb = (tiles + SORT_WARPS - 1) / SORT_WARPS;
    // Pass p reads what pass p - 1 wrote (pass 0: the caller's keys, value = index) and writes the caller's outputs
    // when an even number of passes follows it, else the scratch copy: the last pass always lands in the outputs and
    // the input is never written.  Nothing in the scratch has to start at zero: every word a pass reads was written
    // earlier in the same call (hist and total by k_radix_hist / k_radix_scan for all `tiles` sub-tiles and 256
    // digits, keys / vals by the pass before); what an earlier call left behind is never read.
    const unsigned *kin = cell;
    const int *vin = nullptr;
    for (int p = 0; p < passes; ++p) {
        const bool to_out = ((passes - 1 - p) & 1) == 0;
        unsigned *kout = to_out ? cell_sorted : sc->keys;
        int *vout = to_out ? perm : sc->vals;
        k_radix_hist<<<sb, SORT_BLOCK, 0, s>>>(kin, n, ipw, tiles, 8 * p, sc->hist);
        k_radix_scan<<<RADIX, SORT_BLOCK, 0, s>>>(sc->hist, tiles, sc->total);
        k_radix_scatter<<<sb, SORT_BLOCK, 0, s>>>(kin, vin, kout, vout, n, ipw, tiles, 8 * p, sc->hist, sc->total);
        kin = kout; vin = vout;
    }
    CK(cudaGetLastError());
    return LBM_OK;
}

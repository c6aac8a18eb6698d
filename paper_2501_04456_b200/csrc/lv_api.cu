// lv_api.cu -- the C ABI of include/lv.h: host-side handle, derivation of the
// fp32 tables (fp64 -> fp32 once), workspace carving, CUDA-graph capture of one
// step and the state / debug accessors.  Every step of the path runs in the
// kernels of lv_kernels.cu / lv_sort.cu; there is no CPU fallback.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "lv_internal.cuh"

struct lv_sim {
    int n = 0, n_types = 0;
    uint64_t seed = 0;
    double dt = 0.0;
    bool types_set = false, sched_set = false, bound = false, state_set = false;
    // counting mode: keys, arrival ranks and the cell histogram of the CURRENT posA are in
    // place (written by lv_set_state's first step or by the previous step's update kernel)
    bool hashed = false;
    // skin neighbour list (lv_set_neighbour_list); list_cap = 0: off
    double skin = 0.0;
    int list_cap = 0;               // 0: off; > 0: pool of list_cap entries per NP; -1: automatic pool
    // slot order of `force`: B (ids in velB) after lv_compute_forces, A after lv_step
    bool force_order_b = true;
    lv_type types[LV_MAX_TYPES];
    double eps[LV_MAX_TYPES * LV_MAX_TYPES];
    double sig[LV_MAX_TYPES * LV_MAX_TYPES];
    double rcut[LV_MAX_TYPES * LV_MAX_TYPES];
    double coulomb_k = 0.0;
    double g = 0.0;
    double om2[3] = {0.0, 0.0, 0.0};
    int wall_mode = LV_WALL_ONESIDED;
    int sched_mode = LV_SCHED_CONST;
    double R0 = 0.0, R1 = 0.0;
    int64_t sched_steps = 0;
    int32_t cells_per_cut[LV_MAX_TYPES];
    int sort_mode = LV_SORT_COUNTING;
    int force_kernel = LV_FORCE_SEGMENTS;
    int tile_substreams = 4;        // LV_OPT_TILE_SUBSTREAMS: lanes per target of LV_FORCE_TILE
    int list_lanes = 0;             // LV_OPT_LIST_LANES: lanes per NP of the list force kernel (0: automatic)
    int tile_span = -1;             // LV_OPT_TILE_SPAN: cells along x a tile may span beyond its first (-1: k_a - 1)
    lv_grid_info grid;
    int sort_end_bit = 1;
    size_t ws_bytes = 0;
    LvDev dev;
    LvBufs bufs;
    cudaStream_t stream = nullptr;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t graph_exec = nullptr;
    int launches_per_step = 0;
    // stage timing (measurement aid): (LV_N_STAGES + 1) events per step
    cudaEvent_t *tim_ev = nullptr;
    int tim_cap = 0, tim_used = 0;
    char cuda_err[256];
};

namespace {

constexpr size_t kAlign = 256;
inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

int cuda_fail(lv_sim *s, cudaError_t e, const char *where)
{
    snprintf(s->cuda_err, sizeof(s->cuda_err), "%s: %s", where, cudaGetErrorString(e));
    return LV_E_CUDA;
}
#define LV_CUDA(s, call)                                        \
    do {                                                        \
        cudaError_t e_ = (call);                                \
        if (e_ != cudaSuccess) return cuda_fail((s), e_, #call); \
    } while (0)

// DESIGN.md "Grid rule" (restated independently of the oracle): one grid per NP
// type b, h_b = r_c,bb (1 + 2^-9) / k_b, covering the largest droplet plus one
// largest NP diameter; stencil half-width w_ab = ceil(r_c,ab (1 + 2^-10) / h_b).
int derive_grid(lv_sim *s)
{
    const int T = s->n_types;
    const double Rmax = s->sched_mode == LV_SCHED_CONST ? s->R0 : std::fmax(s->R0, s->R1);
    double smax = 0.0;
    for (int a = 0; a < T; ++a) smax = std::fmax(smax, s->types[a].sigma);
    lv_grid_info &g = s->grid;
    memset(&g, 0, sizeof(g));
    g.n_types = T;
    uint64_t base = 0;
    for (int b = 0; b < T; ++b) {
        const double h = s->rcut[b * LV_MAX_TYPES + b] * (1.0 + 1.0 / 512.0) / (double)s->cells_per_cut[b];
        const double Gd = std::ceil((2.0 * Rmax + 2.0 * smax) / h);
        if (!(Gd >= 1.0) || Gd > 1600.0) return LV_E_ARG;
        const int G = (int)Gd;
        g.h[b] = h;
        g.G[b] = G;
        g.lo[b] = (float)(-0.5 * (double)G * h);
        g.inv_h[b] = (float)(1.0 / h);
        g.base[b] = (uint32_t)base;
        base += (uint64_t)G * G * G;
        if (base > (1ull << 30)) return LV_E_ARG;
    }
    g.base[T] = (uint32_t)base;
    for (int a = 0; a < T; ++a)
        for (int b = 0; b < T; ++b) {
            const double w = std::ceil(s->rcut[a * LV_MAX_TYPES + b] * (1.0 + 1.0 / 1024.0) / g.h[b]);
            if (w > 100.0) return LV_E_ARG;
            // the stencil of the skin list (r_c,ab + skin) is kept in an int8 as well
            if (std::ceil((s->rcut[a * LV_MAX_TYPES + b] + s->skin) * (1.0 + 1.0 / 1024.0) / g.h[b]) > 100.0)
                return LV_E_ARG;
            g.w[a * LV_MAX_TYPES + b] = (int32_t)w;
        }
    int bits = 1;
    while (bits < 32 && (1ull << bits) < base) ++bits;
    s->sort_end_bit = bits;
    return LV_OK;
}

struct Layout {
    size_t posA, velA, posB, velB, force, key_in, key_out, val_in, val_out, cell_off, sort_temp,
        sort_temp_bytes, st, staging, cell_cnt, scan_tile, scan_ticket, posP, list, list_cnt,
        list_start, list_len, list_scan_tile, list_scan_ticket, pos_ref, total;
};

// Pool of the skin list in entries: list_cap per NP on average (a crowded NP may use more than
// its share); automatic: 2048 entries per NP, at most 2 GiB.
size_t list_pool_of(const lv_sim *s)
{
    if (s->list_cap == 0) return 0;
    const size_t n = (size_t)(s->n > 0 ? s->n : 1);
    size_t entries = s->list_cap > 0 ? n * (size_t)s->list_cap : n * 2048;
    if (s->list_cap < 0 && entries > ((size_t)1 << 29)) entries = (size_t)1 << 29;
    entries += 64;
    return entries > 0xfffffff0ull ? 0xfffffff0ull : entries;
}

Layout layout_of(const lv_sim *s)
{
    Layout L;
    const size_t n = (size_t)(s->n > 0 ? s->n : 1);
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
    // positions: one slot more, a dummy far outside every cut-off (the padding of the skin lists points at it)
    L.posA = take(16 * (n + 1)); L.velA = take(16 * n);
    L.posB = take(16 * (n + 1)); L.velB = take(16 * n);
    L.force = take(16 * n);
    L.key_in = take(4 * n); L.key_out = take(4 * n);
    L.val_in = take(4 * n); L.val_out = take(4 * n);
    const size_t n_cells1 = (size_t)s->grid.base[s->n_types] + 1;
    L.cell_off = take(4 * n_cells1);
    L.cell_cnt = take(4 * n_cells1);
    L.scan_tile = take(8 * ((n_cells1 + kScanTile - 1) / kScanTile));
    L.scan_ticket = take(4);
    L.sort_temp_bytes = lvs_temp_bytes(s->n, s->sort_end_bit);
    L.sort_temp = take(L.sort_temp_bytes);
    L.st = take(sizeof(LvDevState));
    // host-transfer staging (28 B per NP); also the scratch of the observables, so never
    // smaller than their largest histogram (8 * 8192 + 64 B)
    L.staging = take(28 * n > 65600 ? 28 * n : 65600);
    L.posP = take(16 * (n + 4));   // pair-interleaved copy of posB + dummy slots (LV_FORCE_PACKED)
    L.list = take(4 * list_pool_of(s));
    L.list_cnt = take(s->list_cap != 0 ? 4 * (n + 1) : 0);
    L.list_start = take(s->list_cap != 0 ? 4 * (n + 1) : 0);
    L.list_len = take(s->list_cap != 0 ? 4 * (n + 1) : 0);
    L.list_scan_tile = take(s->list_cap != 0 ? 8 * ((n + 1 + kScanTile - 1) / kScanTile) : 0);
    L.list_scan_ticket = take(4);
    L.pos_ref = take(s->list_cap != 0 ? 16 * n : 0);
    L.total = o;
    return L;
}

void derive_tables(lv_sim *s)
{
    LvDev &d = s->dev;
    memset(&d, 0, sizeof(d));
    const int T = s->n_types;
    d.n = s->n;
    d.n_types = T;
    d.n_cells = s->grid.base[T];
    d.n_scan_tiles = (uint32_t)(((size_t)d.n_cells + 1 + kScanTile - 1) / kScanTile);
    d.wall_mode = s->wall_mode;
    d.list_cap = s->list_cap;
    d.list_pool = (uint32_t)list_pool_of(s);
    d.list_lanes_forced = s->list_lanes;
    d.n_list_tiles = (uint32_t)(((size_t)(s->n > 0 ? s->n : 1) + 1 + kScanTile - 1) / kScanTile);
    d.skin = (float)s->skin;
    {   // rebuild once an NP is farther than half the skin (less 0.1 % for fp32 rounding) from its build position
        const double hs = 0.5 * s->skin * (1.0 - 1e-3);
        d.half_skin2 = (float)(hs * hs);
    }
    for (int a = 0; a < T; ++a)
        for (int b = 0; b < T; ++b) {
            const int k = a * LV_MAX_TYPES + b;
            const double sg = s->sig[k], s6 = sg * sg * sg * sg * sg * sg;
            d.pair[k].rc2 = (float)(s->rcut[k] * s->rcut[k]);
            d.pair[k].c12 = (float)(48.0 * s->eps[k] * s6 * s6);
            d.pair[k].c6 = (float)(24.0 * s->eps[k] * s6);
            d.pair[k].qq = (float)(s->coulomb_k * s->types[a].charge * s->types[b].charge);
            d.w[k] = (int8_t)s->grid.w[k];
            d.wl[k] = (int8_t)std::ceil((s->rcut[k] + s->skin) * (1.0 + 1.0 / 1024.0) / s->grid.h[b]);
        }
    for (int a = 0; a < T; ++a) {
        const lv_type &t = s->types[a];
        d.type[a].dt_over_m = (float)(s->dt / t.mass);
        d.type[a].a = (float)t.drag_a;
        d.type[a].b = (float)t.kick_b;
        d.type[a].mass = (float)t.mass;
        d.type[a].radius = (float)(0.5 * t.sigma);
        d.wall_k_d[a] = t.wall_k;
        d.radius_d[a] = 0.5 * t.sigma;
        d.grid[a].lo = s->grid.lo[a];
        d.grid[a].inv_h = s->grid.inv_h[a];
        d.grid[a].G = s->grid.G[a];
        d.grid[a].base = s->grid.base[a];
    }
    for (int a = 0; a < T; ++a)
        d.tile_cells[a] = s->tile_span >= 0 ? s->tile_span : s->cells_per_cut[a] - 1;
    d.dt = (float)s->dt;
    d.g = (float)s->g;
    for (int k = 0; k < 3; ++k) d.om2[k] = (float)s->om2[k];
    d.sched_mode = s->sched_mode;
    d.sched_steps = s->sched_steps;
    d.R0 = s->R0;
    d.R1 = s->R1;
    d.seed_lo = (uint32_t)s->seed;
    d.seed_hi = (uint32_t)(s->seed >> 32);
}

// The stages of one step, in order (LV_N_STAGES = 5).  Radix mode: hash | CUB radix
// sort | offsets + scatter | pair force | update.  Counting mode (default): hash +
// histogram | scan (= cell offsets) | place + rank/gather | pair force | update.
int enqueue_stage(lv_sim *s, int stage, bool list_step = false)
{
    const bool counting = s->sort_mode == LV_SORT_COUNTING;
    if (list_step) {
        // Skin-list step (lv_set_neighbour_list; counting sort only).  Stages 0-2 are the same
        // rebuild kernels, each returning at once unless the device-side flag of this step is
        // raised, plus the list build; stages 3-4 work in the list's slot order.
        switch (stage) {
        case 0: LV_CUDA(s, lvk_hash_count(s->dev, s->bufs, true, s->stream)); break;
        case 1: LV_CUDA(s, lvk_scan_cells(s->dev, s->bufs, true, s->stream)); break;
        case 2:
            LV_CUDA(s, lvk_place(s->dev, s->bufs, true, s->stream));
            LV_CUDA(s, lvk_rank_gather(s->dev, s->bufs, false, true, s->stream));
            LV_CUDA(s, lvk_list_build(s->dev, s->bufs, s->stream));
            // the cell kernel of a step whose list does not fit (or is deferred): such a step
            // always rebuilds the cells, so the kernel sits with the rebuild chain -- inside the
            // IF node of the step graph -- and an ordinary step does not launch it at all
            LV_CUDA(s, lvk_pair_force_fallback(s->dev, s->bufs, s->stream));
            break;
        case 3:
            LV_CUDA(s, lvk_pair_force_list(s->dev, s->bufs, s->stream));
            break;
        default: LV_CUDA(s, lvk_update_list(s->dev, s->bufs, s->stream)); break;
        }
        return LV_OK;
    }
    switch (stage) {
    case 0:
        if (counting) {
            // steady state: the previous step's update kernel has already hashed posA
            if (!s->hashed) LV_CUDA(s, lvk_hash_count(s->dev, s->bufs, false, s->stream));
            s->hashed = true;
        } else {
            LV_CUDA(s, lvk_hash(s->dev, s->bufs, s->stream));
        }
        break;
    case 1:
        if (counting) { LV_CUDA(s, lvk_scan_cells(s->dev, s->bufs, false, s->stream)); s->hashed = false; }
        else LV_CUDA(s, lvs_sort_pairs(s->bufs.sort_temp, s->bufs.sort_temp_bytes, s->bufs.key_in,
                                       s->bufs.key_out, s->bufs.val_in, s->bufs.val_out, s->n,
                                       s->sort_end_bit, s->stream));
        break;
    case 2:
        if (counting) {
            LV_CUDA(s, lvk_place(s->dev, s->bufs, false, s->stream));
            LV_CUDA(s, lvk_rank_gather(s->dev, s->bufs, s->force_kernel == LV_FORCE_PACKED || s->force_kernel == LV_FORCE_TILE, false, s->stream));
        } else {
            LV_CUDA(s, lvk_bounds_scatter(s->dev, s->bufs, s->force_kernel == LV_FORCE_PACKED || s->force_kernel == LV_FORCE_TILE, s->stream));
        }
        break;
    case 3:
        if (s->force_kernel == LV_FORCE_TILE)
            LV_CUDA(s, lvk_pair_force_tile(s->dev, s->bufs, s->tile_substreams, lvk_any_charge(s->dev), s->stream));
        else
            LV_CUDA(s, lvk_pair_force(s->dev, s->bufs, s->force_kernel, s->stream));
        break;
    default:
        LV_CUDA(s, lvk_update(s->dev, s->bufs, counting, s->stream));
        s->hashed = counting;
        break;
    }
    return LV_OK;
}

// steps (i)-(ii): cell rebuild -> pair force
int enqueue_rebuild_and_forces(lv_sim *s)
{
    for (int k = 0; k < 4; ++k) {
        int rc = enqueue_stage(s, k);
        if (rc != LV_OK) return rc;
    }
    return LV_OK;
}

int enqueue_step(lv_sim *s)
{
    if (s->list_cap != 0) {
        for (int k = 0; k < LV_N_STAGES; ++k) {
            int rc = enqueue_stage(s, k, true);
            if (rc != LV_OK) return rc;
        }
        return LV_OK;
    }
    int rc = enqueue_rebuild_and_forces(s);
    if (rc != LV_OK) return rc;
    return enqueue_stage(s, 4);
}

// One step as direct launches with an event before the first and after each stage.
int enqueue_step_timed(lv_sim *s, cudaEvent_t *ev)
{
    LV_CUDA(s, cudaEventRecord(ev[0], s->stream));
    for (int k = 0; k < LV_N_STAGES; ++k) {
        int rc = enqueue_stage(s, k, s->list_cap != 0);
        if (rc != LV_OK) return rc;
        LV_CUDA(s, cudaEventRecord(ev[k + 1], s->stream));
    }
    return LV_OK;
}

void free_timing(lv_sim *s)
{
    if (s->tim_ev) {
        for (int k = 0; k < s->tim_cap * (LV_N_STAGES + 1); ++k)
            if (s->tim_ev[k]) cudaEventDestroy(s->tim_ev[k]);
        free(s->tim_ev);
    }
    s->tim_ev = nullptr;
    s->tim_cap = s->tim_used = 0;
}

// Capture one step into a graph (nothing executes during capture).  The graph
// is static: the step index and the radius live in device memory.
// List step as a graph with an IF node: [condition kernel] -> IF(rebuild flag){ rebuild chain:
// stages 0..2 } -> list force, cell force (guarded) -> update.  The body is captured on a
// helper stream into the conditional node's body graph.
// `s->stream` is capturing into graph `g` (as the origin or joined to it): append one list step.
int enqueue_list_step_if(lv_sim *s, cudaGraph_t g, cudaGraph_t *body_out)
{
    cudaGraphConditionalHandle h;
    LV_CUDA(s, cudaGraphConditionalHandleCreate(&h, g, 0, 0));
    int rc = LV_OK;
    cudaError_t e = lvk_list_cond((unsigned long long)h, s->bufs, s->stream);
    cudaStream_t helper = nullptr;
    if (e == cudaSuccess) {
        cudaStreamCaptureStatus cst;
        const cudaGraphNode_t *deps = nullptr;
        size_t nd = 0;
        cudaGraph_t cg = nullptr;
        e = cudaStreamGetCaptureInfo_v2(s->stream, &cst, nullptr, &cg, &deps, &nd);
        cudaGraphNodeParams np = {};
        np.type = cudaGraphNodeTypeConditional;
        np.conditional.handle = h;
        np.conditional.type = cudaGraphCondTypeIf;
        np.conditional.size = 1;
        cudaGraphNode_t cn = nullptr;
        if (e == cudaSuccess) e = cudaGraphAddNode(&cn, cg, deps, nd, &np);
        if (e == cudaSuccess) e = cudaStreamUpdateCaptureDependencies(s->stream, &cn, 1, cudaStreamSetCaptureDependencies);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&helper, cudaStreamNonBlocking);
        if (e == cudaSuccess) {
            cudaGraph_t body = np.conditional.phGraph_out[0];
            if (body_out) *body_out = body;
            e = cudaStreamBeginCaptureToGraph(helper, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed);
            if (e == cudaSuccess) {
                cudaStream_t keep = s->stream;
                s->stream = helper;                 // the stage functions launch on s->stream
                for (int k = 0; k < 3 && rc == LV_OK; ++k) rc = enqueue_stage(s, k, true);
                s->stream = keep;
                cudaGraph_t tmp = nullptr;
                cudaError_t e2 = cudaStreamEndCapture(helper, &tmp);
                if (e == cudaSuccess) e = e2;
            }
        }
    }
    for (int k = 3; k < LV_N_STAGES && rc == LV_OK && e == cudaSuccess; ++k) rc = enqueue_stage(s, k, true);
    if (helper) cudaStreamDestroy(helper);
    if (rc != LV_OK) return rc;
    if (e != cudaSuccess) return cuda_fail(s, e, "capture of the list step");
    return LV_OK;
}

int capture_list_step(lv_sim *s, cudaGraph_t g, cudaGraph_t *body_out)
{
    LV_CUDA(s, cudaStreamBeginCaptureToGraph(s->stream, g, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed));
    int rc = enqueue_list_step_if(s, g, body_out);
    cudaGraph_t gout = nullptr;
    cudaError_t e3 = cudaStreamEndCapture(s->stream, &gout);
    if (rc != LV_OK) return rc;
    if (e3 != cudaSuccess) return cuda_fail(s, e3, "cudaStreamEndCapture");
    return LV_OK;
}

// Capture one step into a graph (nothing executes during capture).  The graph
// is static: the step index and the radius live in device memory.
int build_graph(lv_sim *s)
{
    if (s->stream == nullptr || s->n == 0) return LV_OK;   // legacy stream: direct launches
    cudaGraph_t g = nullptr, body = nullptr;
    int rc = LV_OK;
    if (s->list_cap != 0) {
        LV_CUDA(s, cudaGraphCreate(&g, 0));
        rc = capture_list_step(s, g, &body);
        if (rc != LV_OK) { cudaGraphDestroy(g); return rc; }
    } else {
        LV_CUDA(s, cudaStreamBeginCapture(s->stream, cudaStreamCaptureModeRelaxed));
        s->hashed = s->sort_mode == LV_SORT_COUNTING;      // the graph is the steady-state step
        rc = enqueue_step(s);
        s->hashed = false;
        cudaError_t e = cudaStreamEndCapture(s->stream, &g);
        if (rc != LV_OK) { if (g) cudaGraphDestroy(g); return rc; }     // the capture has been ended above
        if (e != cudaSuccess) return cuda_fail(s, e, "cudaStreamEndCapture");
    }
    s->graph = g;
    // kernels of one step (the IF node's body included)
    int kernels = 0;
    cudaError_t e2 = cudaSuccess;
    {
        cudaGraph_t todo[2] = {g, body};
        for (int q = 0; q < 2 && todo[q] && e2 == cudaSuccess; ++q) {
            size_t nn = 0;
            e2 = cudaGraphGetNodes(todo[q], nullptr, &nn);
            cudaGraphNode_t *nodes = (cudaGraphNode_t *)malloc(sizeof(cudaGraphNode_t) * (nn ? nn : 1));
            if (!nodes) { cudaGraphDestroy(g); s->graph = nullptr; return LV_E_NOMEM; }
            if (e2 == cudaSuccess) e2 = cudaGraphGetNodes(todo[q], nodes, &nn);
            for (size_t i = 0; e2 == cudaSuccess && i < nn; ++i) {
                cudaGraphNodeType t;
                if (cudaGraphNodeGetType(nodes[i], &t) != cudaSuccess) {
                    (void)cudaGetLastError();       // the conditional node: not a kernel; leave no stale error behind
                    continue;
                }
                if (t == cudaGraphNodeTypeKernel) ++kernels;
            }
            free(nodes);
        }
    }
    (void)cudaGetLastError();
    if (e2 == cudaSuccess) e2 = cudaGraphInstantiate(&s->graph_exec, g, 0);
    if (e2 != cudaSuccess) {          // leave no half-built graph behind
        cudaGraphDestroy(g);
        s->graph = nullptr;
        s->graph_exec = nullptr;
        return cuda_fail(s, e2, "cudaGraphGetNodes / cudaGraphInstantiate");
    }
    s->launches_per_step = kernels;
    return LV_OK;
}

int copy_out(lv_sim *s, void *dst, const void *src_dev, size_t bytes, int on_device)
{
    LV_CUDA(s, cudaMemcpyAsync(dst, src_dev, bytes,
                               on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, s->stream));
    return LV_OK;
}

}  // namespace

extern "C" {

int lv_langevin_coeffs(double gamma, double kT, double mass, double dt, double *a, double *b)
{
    if (!a || !b || !(mass > 0.0) || !(dt > 0.0) || !(kT >= 0.0) || !(gamma >= 0.0)) return LV_E_ARG;
    *a = 1.0 - gamma * dt;
    *b = std::sqrt((kT / mass) * (1.0 - (*a) * (*a)));
    return LV_OK;
}

int lv_create(lv_sim **out, int n, int n_types, uint64_t seed, double dt)
{
    if (!out || n < 0 || n >= (1 << 28) || n_types < 1 || n_types > LV_MAX_TYPES || !(dt > 0.0)) return LV_E_ARG;
    lv_sim *s = new (std::nothrow) lv_sim();
    if (!s) return LV_E_NOMEM;
    s->n = n;
    s->n_types = n_types;
    s->seed = seed;
    s->dt = dt;
    for (int b = 0; b < LV_MAX_TYPES; ++b) s->cells_per_cut[b] = 1;
    s->cuda_err[0] = 0;
    memset(&s->bufs, 0, sizeof(s->bufs));
    *out = s;
    return LV_OK;
}

int lv_set_types(lv_sim *s, int n_types, const lv_type *types, const double *eps_TxT,
                 const double *sigma_TxT, const double *rcut_TxT, double cut_factor, double coulomb_k)
{
    if (!s || !types || n_types != s->n_types) return LV_E_ARG;
    if (s->bound) return LV_E_ORDER;
    const int T = n_types;
    for (int a = 0; a < T; ++a) {
        const lv_type &t = types[a];
        if (!(t.sigma > 0.0) || !(t.mass > 0.0) || !(t.wall_k >= 0.0) || !(t.kick_b >= 0.0) ||
            !std::isfinite(t.charge) || !std::isfinite(t.drag_a) || !(t.eps >= 0.0))
            return LV_E_ARG;
    }
    if (!rcut_TxT && !(cut_factor > 0.0)) return LV_E_ARG;
    for (int a = 0; a < T; ++a)
        for (int b = 0; b < T; ++b) {
            const int k = a * LV_MAX_TYPES + b, u = a * T + b, ut = b * T + a;
            const double sg = sigma_TxT ? sigma_TxT[u] : 0.5 * types[a].sigma + 0.5 * types[b].sigma;
            const double ep = eps_TxT ? eps_TxT[u] : std::sqrt(types[a].eps * types[b].eps);
            const double rc = rcut_TxT ? rcut_TxT[u] : cut_factor * sg;
            if (!(sg > 0.0) || !(ep >= 0.0) || !(rc > 0.0)) return LV_E_ARG;
            if ((sigma_TxT && sigma_TxT[u] != sigma_TxT[ut]) || (eps_TxT && eps_TxT[u] != eps_TxT[ut]) ||
                (rcut_TxT && rcut_TxT[u] != rcut_TxT[ut]))
                return LV_E_ARG;
            s->sig[k] = sg;
            s->eps[k] = ep;
            s->rcut[k] = rc;
        }
    memcpy(s->types, types, sizeof(lv_type) * T);
    s->coulomb_k = coulomb_k;
    s->types_set = true;
    return LV_OK;
}

int lv_set_forces(lv_sim *s, double g, const double *omega2_xyz, int wall_mode)
{
    if (!s || !std::isfinite(g) || (wall_mode != LV_WALL_ONESIDED && wall_mode != LV_WALL_WINDOW))
        return LV_E_ARG;
    if (s->bound) return LV_E_ORDER;
    s->g = g;
    for (int k = 0; k < 3; ++k) s->om2[k] = omega2_xyz ? omega2_xyz[k] : 0.0;
    s->wall_mode = wall_mode;
    return LV_OK;
}

int lv_set_droplet_schedule(lv_sim *s, int mode, double R0, double R1, int64_t n_steps)
{
    if (!s || mode < LV_SCHED_CONST || mode > LV_SCHED_R2LAW || !(R0 > 0.0)) return LV_E_ARG;
    if (mode != LV_SCHED_CONST && (!(R1 > 0.0) || n_steps < 1)) return LV_E_ARG;
    if (s->bound) return LV_E_ORDER;
    s->sched_mode = mode;
    s->R0 = R0;
    s->R1 = mode == LV_SCHED_CONST ? R0 : R1;
    s->sched_steps = mode == LV_SCHED_CONST ? 0 : n_steps;
    s->sched_set = true;
    return LV_OK;
}

int lv_set_grid(lv_sim *s, const int32_t *cells_per_cut)
{
    if (!s || !cells_per_cut) return LV_E_ARG;
    if (s->bound) return LV_E_ORDER;
    for (int b = 0; b < s->n_types; ++b)
        if (cells_per_cut[b] < 1 || cells_per_cut[b] > 16) return LV_E_ARG;
    for (int b = 0; b < s->n_types; ++b) s->cells_per_cut[b] = cells_per_cut[b];
    return LV_OK;
}

int lv_set_option(lv_sim *s, int option, int value)
{
    if (!s) return LV_E_ARG;
    if (s->bound) return LV_E_ORDER;
    switch (option) {
    case LV_OPT_SORT:
        if (value != LV_SORT_COUNTING && value != LV_SORT_RADIX) return LV_E_ARG;
        s->sort_mode = value;
        return LV_OK;
    case LV_OPT_FORCE_KERNEL:
        if (value < LV_FORCE_SIMPLE || value > LV_FORCE_TILE) return LV_E_ARG;
        s->force_kernel = value;
        return LV_OK;
    case LV_OPT_TILE_SUBSTREAMS:
        if (value < 1 || value > 32 || (value & (value - 1)) != 0) return LV_E_ARG;
        s->tile_substreams = value;
        return LV_OK;
    case LV_OPT_LIST_LANES:
        if (value < 0 || value > 32 || (value & (value - 1)) != 0) return LV_E_ARG;
        s->list_lanes = value;
        return LV_OK;
    case LV_OPT_TILE_SPAN:
        if (value < -1 || value > 1024) return LV_E_ARG;
        s->tile_span = value;
        return LV_OK;
    default:
        return LV_E_ARG;
    }
}

int lv_set_neighbour_list(lv_sim *s, double skin, int capacity)
{
    if (!s || !std::isfinite(skin) || capacity < -1 || capacity > (1 << 16)) return LV_E_ARG;
    if (s->bound) return LV_E_ORDER;
    // automatic skin: 0.16 of the smallest cut-off (measured on C2 .. C5: a rebuild every ~25 steps
    // instead of ~16 at a tenth pays for the ~8 % longer lists, in the dilute and in the dense states)
    if (capacity != 0 && !(skin > 0.0)) {
        if (!s->types_set) return LV_E_ORDER;
        double rmin = s->rcut[0];
        for (int a = 0; a < s->n_types; ++a)
            for (int b = 0; b < s->n_types; ++b) rmin = std::fmin(rmin, s->rcut[a * LV_MAX_TYPES + b]);
        skin = 0.16 * rmin;
    }
    s->skin = capacity != 0 ? skin : 0.0;
    s->list_cap = capacity;
    return LV_OK;
}

int lv_get_list_stats(lv_sim *s, int64_t *out6)
{
    int64_t *out4 = out6;
    if (!s || !out6) return LV_E_ARG;
    if (!s->bound) return LV_E_ORDER;
    LvDevState h;
    LV_CUDA(s, cudaMemcpyAsync(&h, s->bufs.st, sizeof(h), cudaMemcpyDeviceToHost, s->stream));
    LV_CUDA(s, cudaStreamSynchronize(s->stream));
    out4[0] = (int64_t)h.n_rebuilds;
    out4[1] = (int64_t)h.list_used;
    out4[2] = (int64_t)h.n_fallback;
    out4[3] = (int64_t)s->dev.list_pool;
    out6[4] = (int64_t)h.n_exact;
    out6[5] = (int64_t)h.list_lanes;
    return LV_OK;
}

int lv_get_rebuild_count(lv_sim *s, int64_t *rebuilds)
{
    if (!s || !rebuilds) return LV_E_ARG;
    if (!s->bound) return LV_E_ORDER;
    LvDevState h;
    LV_CUDA(s, cudaMemcpyAsync(&h, s->bufs.st, sizeof(h), cudaMemcpyDeviceToHost, s->stream));
    LV_CUDA(s, cudaStreamSynchronize(s->stream));
    *rebuilds = (int64_t)h.n_rebuilds;
    return LV_OK;
}

size_t lv_workspace_bytes(const lv_sim *cs)
{
    lv_sim *s = const_cast<lv_sim *>(cs);
    if (!s || !s->types_set || !s->sched_set) return 0;
    if (derive_grid(s) != LV_OK) return 0;
    if (s->list_cap == -1 && s->n < 16384) {       // as lv_bind will decide
        lv_sim t = *s;
        t.list_cap = 0;
        return layout_of(&t).total;
    }
    return layout_of(s).total;
}

int lv_bind(lv_sim *s, void *workspace_dev, size_t workspace_bytes, void *cuda_stream)
{
    if (!s) return LV_E_ARG;
    if (!s->types_set || !s->sched_set) return LV_E_ORDER;
    if (s->bound) return LV_E_ORDER;
    // automatic list: a small droplet is bound by launch latency, and the list step has more
    // (mostly idle) launches than the cell step -- keep the cells there
    if (s->list_cap == -1 && s->n < 16384) { s->list_cap = 0; s->skin = 0.0; }
    if (s->list_cap != 0 && s->sort_mode != LV_SORT_COUNTING) return LV_E_ARG;
    int rc = derive_grid(s);
    if (rc != LV_OK) return rc;
    const Layout L = layout_of(s);
    if (!workspace_dev || workspace_bytes < L.total || ((uintptr_t)workspace_dev % kAlign) != 0)
        return LV_E_WORKSPACE;
    unsigned char *w = (unsigned char *)workspace_dev;
    LvBufs &B = s->bufs;
    B.posA = (float4 *)(w + L.posA); B.velA = (float4 *)(w + L.velA);
    B.posB = (float4 *)(w + L.posB); B.velB = (float4 *)(w + L.velB);
    B.force = (float4 *)(w + L.force);
    B.key_in = (uint32_t *)(w + L.key_in); B.key_out = (uint32_t *)(w + L.key_out);
    B.val_in = (uint32_t *)(w + L.val_in); B.val_out = (uint32_t *)(w + L.val_out);
    B.cell_off = (uint32_t *)(w + L.cell_off);
    B.sort_temp = w + L.sort_temp;
    B.sort_temp_bytes = L.sort_temp_bytes;
    B.st = (LvDevState *)(w + L.st);
    B.staging = w + L.staging;
    B.cell_cnt = (uint32_t *)(w + L.cell_cnt);
    B.scan_tile = (unsigned long long *)(w + L.scan_tile);
    B.scan_ticket = (unsigned int *)(w + L.scan_ticket);
    B.posP = (float *)(w + L.posP);
    B.list = (uint32_t *)(w + L.list);
    B.list_cnt = (uint32_t *)(w + L.list_cnt);
    B.list_start = (uint32_t *)(w + L.list_start);
    B.list_len = (uint32_t *)(w + L.list_len);
    B.list_scan_tile = (unsigned long long *)(w + L.list_scan_tile);
    B.list_scan_ticket = (unsigned int *)(w + L.list_scan_ticket);
    B.pos_ref = (float4 *)(w + L.pos_ref);
    s->ws_bytes = L.total;
    s->stream = (cudaStream_t)cuda_stream;
    derive_tables(s);
    LV_CUDA(s, lvk_tile_prepare());
    LV_CUDA(s, cudaMemsetAsync(B.st, 0, sizeof(LvDevState), s->stream));
    // the histogram is zero between steps: the scan clears what it has read
    LV_CUDA(s, cudaMemsetAsync(B.cell_cnt, 0, 4 * ((size_t)s->grid.base[s->n_types] + 1), s->stream));
    rc = build_graph(s);
    if (rc != LV_OK) return rc;
    s->bound = true;
    return LV_OK;
}

int lv_set_state(lv_sim *s, const float *pos_xyz, const float *vel_xyz, const int32_t *type,
                 int64_t step, int on_device)
{
    if (!s || step < 0) return LV_E_ARG;
    if (!s->bound) return LV_E_ORDER;
    if (s->n > 0 && (!pos_xyz || !vel_xyz || !type)) return LV_E_ARG;
    const size_t n = (size_t)s->n;
    const float *dp = pos_xyz, *dv = vel_xyz;
    const int32_t *dt = type;
    if (!on_device && n > 0) {
        unsigned char *stg = s->bufs.staging;
        LV_CUDA(s, cudaMemcpyAsync(stg, pos_xyz, 12 * n, cudaMemcpyHostToDevice, s->stream));
        LV_CUDA(s, cudaMemcpyAsync(stg + 12 * n, vel_xyz, 12 * n, cudaMemcpyHostToDevice, s->stream));
        LV_CUDA(s, cudaMemcpyAsync(stg + 24 * n, type, 4 * n, cudaMemcpyHostToDevice, s->stream));
        dp = (const float *)stg;
        dv = (const float *)(stg + 12 * n);
        dt = (const int32_t *)(stg + 24 * n);
    }
    LV_CUDA(s, lvk_pack_state(s->dev, s->bufs, dp, dv, dt, (long long)step, s->stream));
    if (s->hashed) {     // a histogram of the replaced state is pending: clear it
        LV_CUDA(s, cudaMemsetAsync(s->bufs.cell_cnt, 0, 4 * ((size_t)s->grid.base[s->n_types] + 1),
                                   s->stream));
        s->hashed = false;
    }
    if (!on_device) LV_CUDA(s, cudaStreamSynchronize(s->stream));
    s->state_set = true;
    return LV_OK;
}

int lv_step(lv_sim *s, int n)
{
    if (!s || n < 0) return LV_E_ARG;
    if (!s->bound || !s->state_set) return LV_E_ORDER;
    if (s->n == 0) return LV_OK;
    // after the update kernel A has the slot order of `force`; in list mode B may be stale
    if (n > 0) s->force_order_b = false;
    if (s->tim_cap > 0) {
        if (n > s->tim_cap - s->tim_used) return LV_E_ARG;
        for (int k = 0; k < n; ++k) {
            int rc = enqueue_step_timed(s, s->tim_ev + (size_t)s->tim_used * (LV_N_STAGES + 1));
            if (rc != LV_OK) return rc;
            ++s->tim_used;
        }
        return LV_OK;
    }
    for (int k = 0; k < n; ++k) {
        if (s->graph_exec) {
            if (s->sort_mode == LV_SORT_COUNTING && s->list_cap == 0 && !s->hashed) {
                LV_CUDA(s, lvk_hash_count(s->dev, s->bufs, false, s->stream));
                s->hashed = true;        // and the graph's update kernel leaves it true
            }
            LV_CUDA(s, cudaGraphLaunch(s->graph_exec, s->stream));
        } else {
            int rc = enqueue_step(s);
            if (rc != LV_OK) return rc;
        }
    }
    return LV_OK;
}

int lv_compute_forces(lv_sim *s)
{
    if (!s) return LV_E_ARG;
    if (!s->bound || !s->state_set) return LV_E_ORDER;
    if (s->n == 0) return LV_OK;
    s->force_order_b = true;
    return enqueue_rebuild_and_forces(s);
}

namespace {
constexpr int kMaxObsBins = 8192;

// scratch for the observables: the host-transfer staging area (28 n bytes)
int obs_scratch(lv_sim *s, int n_bins, unsigned long long **hist, double **sums)
{
    const size_t need = 8 * (size_t)n_bins + 64;
    const size_t have = 28 * (size_t)s->n > 65600 ? 28 * (size_t)s->n : 65600;
    if (need > have) return LV_E_ARG;
    *hist = (unsigned long long *)s->bufs.staging;
    *sums = (double *)(s->bufs.staging + 8 * (size_t)n_bins);
    LV_CUDA(s, cudaMemsetAsync(s->bufs.staging, 0, need, s->stream));
    return LV_OK;
}

double shell_volume(int k, double dr)
{
    const double a = k * dr, b = (k + 1) * dr;
    return 4.0 / 3.0 * M_PI * (b * b * b - a * a * a);
}
}  // namespace

int lv_observe_rdf(lv_sim *s, double dr, int n_bins, uint64_t *hist, double *g)
{
    if (!s || !(dr > 0.0) || n_bins < 1 || n_bins > kMaxObsBins) return LV_E_ARG;
    if (!s->bound || !s->state_set) return LV_E_ORDER;
    if (hist) memset(hist, 0, 8 * (size_t)n_bins);
    if (g) for (int k = 0; k < n_bins; ++k) g[k] = 0.0;
    for (int b = 0; b < s->n_types; ++b)       // the pair walk keeps its stencil half-width in an int8
        if (std::ceil(dr * (double)n_bins * (1.0 + 1.0 / 1024.0) / s->grid.h[b]) > 100.0) return LV_E_ARG;
    if (s->n == 0) return LV_OK;
    // cell structures of the current state (steps (i) of PAPER.md:64), then the pair walk
    for (int k = 0; k < 3; ++k) {
        int rc = enqueue_stage(s, k);
        if (rc != LV_OK) return rc;
    }
    unsigned long long *dh = nullptr;
    double *ds = nullptr;
    int rc = obs_scratch(s, n_bins, &dh, &ds);
    if (rc != LV_OK) return rc;
    LV_CUDA(s, lvk_rdf_hist(s->dev, s->bufs, s->grid.h, dr, n_bins, dh, s->stream));
    uint64_t *hh = (uint64_t *)malloc(8 * (size_t)n_bins);
    if (!hh) return LV_E_NOMEM;
    cudaError_t e = cudaMemcpyAsync(hh, dh, 8 * (size_t)n_bins, cudaMemcpyDeviceToHost, s->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
    if (e != cudaSuccess) { free(hh); return cuda_fail(s, e, "lv_observe_rdf"); }
    LvDevState st;
    e = cudaMemcpy(&st, s->bufs.st, sizeof(st), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) { free(hh); return cuda_fail(s, e, "lv_observe_rdf"); }
    // Eq. 6: g_k = (psi_k / N) / ((N - 1) dV_k / V), V the droplet volume at this step
    const double R = lv_radius_of(s->sched_mode, s->R0, s->R1, s->sched_steps, st.step);
    const double V = 4.0 / 3.0 * M_PI * R * R * R, N = (double)s->n;
    for (int k = 0; k < n_bins; ++k) {
        if (hist) hist[k] = hh[k];
        if (g && s->n > 1) g[k] = ((double)hh[k] / N) / ((N - 1.0) * shell_volume(k, dr) / V);
    }
    free(hh);
    return LV_OK;
}

int lv_observe_radial(lv_sim *s, double dr, int n_bins, uint64_t *hist, double *conc, double *centre,
                      double *r_g, double *d_f, int64_t *n_surf)
{
    if (!s || !(dr > 0.0) || n_bins < 1 || n_bins > kMaxObsBins) return LV_E_ARG;
    if (!s->bound || !s->state_set) return LV_E_ORDER;
    if (hist) memset(hist, 0, 8 * (size_t)n_bins);
    if (conc) for (int k = 0; k < n_bins; ++k) conc[k] = 0.0;
    if (centre) centre[0] = centre[1] = centre[2] = 0.0;
    if (r_g) *r_g = 0.0;
    if (d_f) *d_f = 0.0;
    if (n_surf) *n_surf = 0;
    if (s->n == 0) return LV_OK;
    LvDevState st;
    LV_CUDA(s, cudaMemcpyAsync(&st, s->bufs.st, sizeof(st), cudaMemcpyDeviceToHost, s->stream));
    LV_CUDA(s, cudaStreamSynchronize(s->stream));
    const double R = lv_radius_of(s->sched_mode, s->R0, s->R1, s->sched_steps, st.step);
    unsigned long long *dh = nullptr;
    double *ds = nullptr;
    int rc = obs_scratch(s, n_bins, &dh, &ds);
    if (rc != LV_OK) return rc;
    LV_CUDA(s, lvk_radial_hist(s->dev, s->bufs, s->grid.h, R, dr, n_bins, dh, ds, s->stream));
    const size_t bytes = 8 * (size_t)n_bins + 64;
    unsigned char *hb = (unsigned char *)malloc(bytes);
    if (!hb) return LV_E_NOMEM;
    cudaError_t e = cudaMemcpyAsync(hb, dh, bytes, cudaMemcpyDeviceToHost, s->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
    if (e != cudaSuccess) { free(hb); return cuda_fail(s, e, "lv_observe_radial"); }
    const uint64_t *hh = (const uint64_t *)hb;
    const double *sm = (const double *)(hb + 8 * (size_t)n_bins);
    const double N = (double)s->n, V = 4.0 / 3.0 * M_PI * R * R * R;
    for (int k = 0; k < n_bins; ++k) {
        if (hist) hist[k] = hh[k];
        if (conc) conc[k] = ((double)hh[k] / N) / (shell_volume(k, dr) / V);      // Eq. 8
    }
    const double cx = sm[0] / N, cy = sm[1] / N, cz = sm[2] / N;                  // Eq. 4
    const double rg2 = sm[3] / N - (cx * cx + cy * cy + cz * cz);                 // Eq. 3
    const double rg = rg2 > 0.0 ? sqrt(rg2) : 0.0;
    if (centre) { centre[0] = cx; centre[1] = cy; centre[2] = cz; }
    if (r_g) *r_g = rg;
    // Eq. 2 solved for D_f with k_f = 1.593 and d_NP the mean NP diameter
    if (d_f && rg > 0.0) *d_f = log(N / 1.593) / log(2.0 * rg / (sm[4] / N));
    if (n_surf) memcpy(n_surf, sm + 5, 8);
    free(hb);
    return LV_OK;
}

int lv_observe_clusters(lv_sim *s, double bond_factor, int32_t *labels, int64_t *n_clusters,
                        double *mean_size, int64_t *largest, uint64_t *log2_hist)
{
    if (!s || !(bond_factor > 0.0)) return LV_E_ARG;
    if (!s->bound || !s->state_set) return LV_E_ORDER;
    if (n_clusters) *n_clusters = 0;
    if (mean_size) *mean_size = 0.0;
    if (largest) *largest = 0;
    if (log2_hist) memset(log2_hist, 0, 8 * 32);
    if (s->n == 0) return LV_OK;
    const int T = s->n_types;
    float rb2[LV_MAX_TYPES * LV_MAX_TYPES];
    memset(rb2, 0, sizeof(rb2));
    for (int a = 0; a < T; ++a)
        for (int b = 0; b < T; ++b) {
            const int k = a * LV_MAX_TYPES + b;
            const double rb = bond_factor * s->sig[k];
            if (rb > s->rcut[k]) return LV_E_ARG;      // bonds are searched inside the force stencil
            rb2[k] = (float)(rb * rb);
        }
    for (int k = 0; k < 3; ++k) {                      // cell structures of the current state
        int rc = enqueue_stage(s, k);
        if (rc != LV_OK) return rc;
    }
    // scratch in the staging area: 3 uint32[n] | int32 labels[n] | 34 u64 statistics
    const size_t n = (size_t)s->n;
    if ((28 * n > 65600 ? 28 * n : 65600) < 16 * n + 34 * 8 + 8) return LV_E_ARG;   // staging >= 65600 B
    uint32_t *scratch = (uint32_t *)s->bufs.staging;
    int32_t *dlab = (int32_t *)(s->bufs.staging + 12 * n);
    unsigned long long *dst = (unsigned long long *)(s->bufs.staging + ((16 * n + 7) / 8) * 8);
    LV_CUDA(s, cudaMemsetAsync(dst, 0, 34 * 8, s->stream));
    LV_CUDA(s, lvk_clusters(s->dev, s->bufs, rb2, s->grid.h, scratch, labels ? dlab : nullptr, dst, s->stream));
    unsigned long long hs[34];
    LV_CUDA(s, cudaMemcpyAsync(hs, dst, sizeof(hs), cudaMemcpyDeviceToHost, s->stream));
    if (labels) LV_CUDA(s, cudaMemcpyAsync(labels, dlab, 4 * n, cudaMemcpyDeviceToHost, s->stream));
    LV_CUDA(s, cudaStreamSynchronize(s->stream));
    if (n_clusters) *n_clusters = (int64_t)hs[0];
    if (largest) *largest = (int64_t)hs[1];
    if (mean_size && hs[0] > 0) *mean_size = (double)n / (double)hs[0];
    if (log2_hist) for (int k = 0; k < 32; ++k) log2_hist[k] = hs[2 + k];
    return LV_OK;
}

int lv_render(lv_sim *s, const lv_view *view, void *zbuf_dev, uint32_t *rgba, int on_device)
{
    if (!s || !view || !zbuf_dev || !rgba) return LV_E_ARG;
    if (view->width < 1 || view->height < 1 || view->width > 8192 || view->height > 8192) return LV_E_ARG;
    if (!(view->eye_dist > 0.0) || !(view->focal_px > 0.0)) return LV_E_ARG;
    if (((uintptr_t)zbuf_dev % 8) != 0) return LV_E_ARG;
    if (!s->bound || !s->state_set) return LV_E_ORDER;
    // rotation = pitch about x after yaw about y, in fp64, rounded once
    const double cy = cos(view->yaw), sy = sin(view->yaw), cp = cos(view->pitch), sp = sin(view->pitch);
    const double m[9] = {cy, 0.0, sy, sp * sy, cp, -sp * cy, -cp * sy, sp, cp * cy};
    float rot[9];
    for (int k = 0; k < 9; ++k) rot[k] = (float)m[k];
    LvDevState st;
    LV_CUDA(s, cudaMemcpyAsync(&st, s->bufs.st, sizeof(st), cudaMemcpyDeviceToHost, s->stream));
    LV_CUDA(s, cudaStreamSynchronize(s->stream));
    const double R = lv_radius_of(s->sched_mode, s->R0, s->R1, s->sched_steps, st.step);
    const size_t n_px = (size_t)view->width * view->height;
    // host output: the image is staged in the caller's scratch, behind the depth keys
    uint32_t *drgba = on_device ? rgba : (uint32_t *)((unsigned long long *)zbuf_dev + n_px);
    cudaError_t e = lvk_render(s->dev, s->bufs, view, rot, R, (unsigned long long *)zbuf_dev, drgba, s->stream);
    if (e == cudaSuccess && !on_device) {
        e = cudaMemcpyAsync(rgba, drgba, 4 * n_px, cudaMemcpyDeviceToHost, s->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
    }
    if (e != cudaSuccess) return cuda_fail(s, e, "lv_render");
    return LV_OK;
}

int lv_render_surface(lv_sim *s, const lv_surface_map *map, void *scratch_dev, uint32_t *rgba,
                      int on_device)
{
    if (!s || !map || !scratch_dev || !rgba) return LV_E_ARG;
    if (map->width < 1 || map->height < 1 || map->width > 8192 || map->height > 8192) return LV_E_ARG;
    if (((uintptr_t)scratch_dev % 8) != 0) return LV_E_ARG;
    if (!s->bound || !s->state_set) return LV_E_ORDER;
    const int W = map->width, H = map->height;
    // direction factors per column / row: fp64 libm, rounded once (include/lv.h)
    struct Tab {                         // freed on every return path
        float *p;
        ~Tab() { free(p); }
    } tabh{(float *)malloc(4 * (2 * (size_t)W + 2 * (size_t)H))};
    float *tab = tabh.p;
    if (!tab) return LV_E_NOMEM;
    for (int px = 0; px < W; ++px) {
        const double lam = -M_PI + (2.0 * M_PI) * (((double)px + 0.5) / (double)W);
        tab[px] = (float)cos(lam);
        tab[W + px] = (float)sin(lam);
    }
    for (int py = 0; py < H; ++py) {
        const double phi = 0.5 * M_PI - M_PI * (((double)py + 0.5) / (double)H);
        tab[2 * W + py] = (float)cos(phi);
        tab[2 * W + H + py] = (float)sin(phi);
    }
    LvDevState st;
    LV_CUDA(s, cudaMemcpyAsync(&st, s->bufs.st, sizeof(st), cudaMemcpyDeviceToHost, s->stream));
    LV_CUDA(s, cudaStreamSynchronize(s->stream));
    const double R = lv_radius_of(s->sched_mode, s->R0, s->R1, s->sched_steps, st.step);
    const size_t n_px = (size_t)W * H;
    unsigned long long *zbuf = (unsigned long long *)scratch_dev;
    float *tab_dev = (float *)(zbuf + n_px);
    LV_CUDA(s, cudaMemcpyAsync(tab_dev, tab, 4 * (2 * (size_t)W + 2 * (size_t)H), cudaMemcpyHostToDevice, s->stream));
    // host output: the image is staged in the caller's scratch, behind the keys and the tables
    uint32_t *drgba = on_device ? rgba : (uint32_t *)(tab_dev + 2 * ((size_t)W + (size_t)H));
    cudaError_t e = lvk_render_surface(s->dev, s->bufs, map, R, tab_dev, zbuf, drgba, s->stream);
    if (e == cudaSuccess && !on_device)
        e = cudaMemcpyAsync(rgba, drgba, 4 * n_px, cudaMemcpyDeviceToHost, s->stream);
    // synchronise in both modes: `tab` is pageable host memory read by the stream
    if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
    if (e != cudaSuccess) return cuda_fail(s, e, "lv_render_surface");
    return LV_OK;
}

int lv_get_status(lv_sim *s, uint32_t *status)
{
    if (!s || !status) return LV_E_ARG;
    if (!s->bound) return LV_E_ORDER;
    LvDevState h;
    LV_CUDA(s, cudaMemcpyAsync(&h, s->bufs.st, sizeof(h), cudaMemcpyDeviceToHost, s->stream));
    LV_CUDA(s, cudaStreamSynchronize(s->stream));
    *status = h.status;
    return LV_OK;
}

int lv_get_state(lv_sim *s, float *pos_xyz, float *vel_xyz, int32_t *type, double *R, int64_t *step,
                 int on_device)
{
    if (!s) return LV_E_ARG;
    if (!s->bound || !s->state_set) return LV_E_ORDER;
    const size_t n = (size_t)s->n;
    if (n > 0 && (pos_xyz || vel_xyz || type)) {
        if (on_device) {
            LV_CUDA(s, lvk_unpack_state(s->dev, s->bufs, pos_xyz, vel_xyz, type, s->stream));
        } else {
            unsigned char *stg = s->bufs.staging;
            float *dp = (float *)stg, *dv = (float *)(stg + 12 * n);
            int32_t *dt = (int32_t *)(stg + 24 * n);
            LV_CUDA(s, lvk_unpack_state(s->dev, s->bufs, pos_xyz ? dp : nullptr, vel_xyz ? dv : nullptr,
                                        type ? dt : nullptr, s->stream));
            if (pos_xyz) LV_CUDA(s, cudaMemcpyAsync(pos_xyz, dp, 12 * n, cudaMemcpyDeviceToHost, s->stream));
            if (vel_xyz) LV_CUDA(s, cudaMemcpyAsync(vel_xyz, dv, 12 * n, cudaMemcpyDeviceToHost, s->stream));
            if (type) LV_CUDA(s, cudaMemcpyAsync(type, dt, 4 * n, cudaMemcpyDeviceToHost, s->stream));
        }
    }
    LvDevState h;
    LV_CUDA(s, cudaMemcpyAsync(&h, s->bufs.st, sizeof(h), cudaMemcpyDeviceToHost, s->stream));
    LV_CUDA(s, cudaStreamSynchronize(s->stream));
    if (step) *step = (int64_t)h.step;
    if (R) *R = lv_radius_of(s->sched_mode, s->R0, s->R1, s->sched_steps, h.step);
    if (h.status & LV_ST_BAD_TYPE) return LV_E_ARG;
    if (h.status & LV_ST_NONFINITE) return LV_E_NONFINITE;
    return LV_OK;          // LV_ST_LIST_OVERFLOW is a warning: those steps ran on the cell kernel
}

int lv_get_forces(lv_sim *s, float *force_xyz, int32_t *neigh_count, int on_device)
{
    if (!s) return LV_E_ARG;
    if (!s->bound || !s->state_set) return LV_E_ORDER;
    const size_t n = (size_t)s->n;
    if (n > 0 && (force_xyz || neigh_count)) {
        if (on_device) {
            LV_CUDA(s, lvk_unpack_forces(s->dev, s->bufs, s->force_order_b, force_xyz, neigh_count, s->stream));
        } else {
            unsigned char *stg = s->bufs.staging;
            float *df = (float *)stg;
            int32_t *dc = (int32_t *)(stg + 12 * n);
            LV_CUDA(s, lvk_unpack_forces(s->dev, s->bufs, s->force_order_b, force_xyz ? df : nullptr,
                                         neigh_count ? dc : nullptr, s->stream));
            if (force_xyz) LV_CUDA(s, cudaMemcpyAsync(force_xyz, df, 12 * n, cudaMemcpyDeviceToHost, s->stream));
            if (neigh_count) LV_CUDA(s, cudaMemcpyAsync(neigh_count, dc, 4 * n, cudaMemcpyDeviceToHost, s->stream));
        }
    }
    LV_CUDA(s, cudaStreamSynchronize(s->stream));
    return LV_OK;
}

int lv_get_debug(lv_sim *s, int what, void *dst, size_t bytes, int on_device)
{
    if (!s || !dst) return LV_E_ARG;
    if (what == LV_DBG_GRID) {   // host-only: available as soon as types and schedule are set
        if (on_device) return LV_E_ARG;
        if (!s->types_set || !s->sched_set) return LV_E_ORDER;
        if (!s->bound) { int rg = derive_grid(s); if (rg != LV_OK) return rg; }
        memcpy(dst, &s->grid, bytes < sizeof(lv_grid_info) ? bytes : sizeof(lv_grid_info));
        return LV_OK;
    }
    if (!s->bound) return LV_E_ORDER;
    const size_t n = (size_t)s->n;
    int rc = LV_OK;
    switch (what) {
    case LV_DBG_KEYS:
        rc = copy_out(s, dst, s->bufs.key_in, bytes < 4 * n ? bytes : 4 * n, on_device); break;
    case LV_DBG_KEYS_SORTED:
        if (s->sort_mode == LV_SORT_COUNTING) {
            if (n == 0) break;
            LV_CUDA(s, lvk_keys_sorted(s->dev, s->bufs, (uint32_t *)s->bufs.staging, s->stream));
            rc = copy_out(s, dst, s->bufs.staging, bytes < 4 * n ? bytes : 4 * n, on_device);
        } else {
            rc = copy_out(s, dst, s->bufs.key_out, bytes < 4 * n ? bytes : 4 * n, on_device);
        }
        break;
    case LV_DBG_PERM:
        rc = copy_out(s, dst, s->bufs.val_out, bytes < 4 * n ? bytes : 4 * n, on_device); break;
    case LV_DBG_CELL_OFFSETS: {
        const size_t full = 4 * ((size_t)s->grid.base[s->n_types] + 1);
        rc = copy_out(s, dst, s->bufs.cell_off, bytes < full ? bytes : full, on_device); break;
    }
    case LV_DBG_IDS_SORTED:
        if (n == 0) break;
        LV_CUDA(s, lvk_ids_sorted(s->dev, s->bufs, (uint32_t *)s->bufs.staging, s->stream));
        rc = copy_out(s, dst, s->bufs.staging, bytes < 4 * n ? bytes : 4 * n, on_device); break;
    default:
        return LV_E_ARG;
    }
    if (rc != LV_OK) return rc;
    LV_CUDA(s, cudaStreamSynchronize(s->stream));
    return LV_OK;
}

int lv_launches_per_step(const lv_sim *s) { return s ? s->launches_per_step : 0; }

int lv_step_profiled(lv_sim *s, float *ms_out)
{
    if (!s || !ms_out) return LV_E_ARG;
    if (!s->bound || !s->state_set) return LV_E_ORDER;
    for (int k = 0; k < LV_N_STAGES; ++k) ms_out[k] = 0.f;
    if (s->n == 0) return LV_OK;
    cudaEvent_t ev[LV_N_STAGES + 1];
    for (int k = 0; k <= LV_N_STAGES; ++k) LV_CUDA(s, cudaEventCreate(&ev[k]));
    int rc = LV_OK;
    cudaError_t e = cudaSuccess;
    e = cudaEventRecord(ev[0], s->stream);
    for (int k = 0; k < LV_N_STAGES && e == cudaSuccess && rc == LV_OK; ++k) {
        rc = enqueue_stage(s, k, s->list_cap != 0);
        if (rc == LV_OK) e = cudaEventRecord(ev[k + 1], s->stream);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
    for (int k = 0; rc == LV_OK && e == cudaSuccess && k < LV_N_STAGES; ++k)
        e = cudaEventElapsedTime(&ms_out[k], ev[k], ev[k + 1]);
    for (int k = 0; k <= LV_N_STAGES; ++k) cudaEventDestroy(ev[k]);
    if (rc == LV_OK && e != cudaSuccess) rc = cuda_fail(s, e, "lv_step_profiled");
    return rc;
}

int lv_stage_timing(lv_sim *s, int capacity)
{
    if (!s || capacity < 0 || capacity > (1 << 20)) return LV_E_ARG;
    if (!s->bound) return LV_E_ORDER;
    LV_CUDA(s, cudaStreamSynchronize(s->stream));
    free_timing(s);
    if (capacity == 0) return LV_OK;
    const size_t ne = (size_t)capacity * (LV_N_STAGES + 1);
    s->tim_ev = (cudaEvent_t *)calloc(ne, sizeof(cudaEvent_t));
    if (!s->tim_ev) return LV_E_NOMEM;
    s->tim_cap = capacity;
    for (size_t k = 0; k < ne; ++k) {
        cudaError_t e = cudaEventCreate(&s->tim_ev[k]);
        if (e != cudaSuccess) { free_timing(s); return cuda_fail(s, e, "cudaEventCreate"); }
    }
    return LV_OK;
}

int lv_read_stage_timing(lv_sim *s, double *ms_stage_sum, double *ms_step_sum, int64_t *steps)
{
    if (!s) return LV_E_ARG;
    if (!s->bound || s->tim_cap == 0) return LV_E_ORDER;
    LV_CUDA(s, cudaStreamSynchronize(s->stream));
    double st[LV_N_STAGES] = {0, 0, 0, 0, 0}, tot = 0.0;
    for (int k = 0; k < s->tim_used; ++k) {
        cudaEvent_t *ev = s->tim_ev + (size_t)k * (LV_N_STAGES + 1);
        float ms = 0.f;
        for (int j = 0; j < LV_N_STAGES; ++j) {
            LV_CUDA(s, cudaEventElapsedTime(&ms, ev[j], ev[j + 1]));
            st[j] += ms;
        }
        LV_CUDA(s, cudaEventElapsedTime(&ms, ev[0], ev[LV_N_STAGES]));
        tot += ms;
    }
    if (ms_stage_sum) for (int j = 0; j < LV_N_STAGES; ++j) ms_stage_sum[j] = st[j];
    if (ms_step_sum) *ms_step_sum = tot;
    if (steps) *steps = s->tim_used;
    s->tim_used = 0;
    return LV_OK;
}

int lv_measure_fp32_peak(void *cuda_stream, void *scratch_dev, double *tflops)
{
    if (!tflops || !scratch_dev) return LV_E_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return LV_E_CUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return LV_E_CUDA;
    float *scratch = (float *)scratch_dev;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    double best = 0.0, flops = 0.0;
    cudaError_t e = cudaSuccess;
    for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {
        cudaEventRecord(e0, st);
        e = lvk_fma_peak(scratch, sms * 8, 4096, &flops, st);
        cudaEventRecord(e1, st);
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e == cudaSuccess && rep > 0 && ms > 0.f) best = std::fmax(best, flops / (ms * 1e-3) * 1e-12);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (e != cudaSuccess) return LV_E_CUDA;
    *tflops = best;
    return LV_OK;
}

int lv_destroy(lv_sim *s)
{
    if (!s) return LV_OK;
    if (s->bound) cudaStreamSynchronize(s->stream);
    if (s->graph_exec) cudaGraphExecDestroy(s->graph_exec);
    if (s->graph) cudaGraphDestroy(s->graph);
    free_timing(s);
    delete s;
    return LV_OK;
}

const char *lv_strerror(int code)
{
    switch (code) {
    case LV_OK: return "ok";
    case LV_E_ARG: return "bad argument";
    case LV_E_ORDER: return "call order violated";
    case LV_E_WORKSPACE: return "workspace too small or misaligned";
    case LV_E_CAPACITY: return "size beyond a fixed maximum of the library (lv_observe_rdf_noalloc: LV_NOALLOC_MAX_BINS)";
    case LV_E_CUDA: return "CUDA runtime error";
    case LV_E_NONFINITE: return "non-finite position or velocity";
    case LV_E_NOMEM: return "host allocation failed";
    default: return "unknown error";
    }
}

const char *lv_last_cuda_error(const lv_sim *s) { return s ? s->cuda_err : ""; }

const char *lv_version(void) { return "lv 0.1.0 (sm_100a)"; }

}  // extern "C"

// ---- batched replicas: R independent lv_sim handles stepped by ONE
// CUDA-graph launch.  The graph holds one step (or `chunk` steps) of every replica as parallel
// branches forked from and joined into the first replica's stream, so the small kernels of
// many small droplets share the GPU without R launch sequences issued from the host.
struct lv_batch {
    int n = 0, chunk = 1;
    lv_sim **sims = nullptr;
    cudaEvent_t *ev = nullptr;          // [n]: join events; ev[0] = fork
    cudaGraph_t graph1 = nullptr, graphk = nullptr;
    cudaGraphExec_t exec1 = nullptr, execk = nullptr;
};

namespace {
// capture `steps` steady-state steps of every replica into one graph
int capture_batch(lv_batch *b, int steps, cudaGraph_t *g, cudaGraphExec_t *x)
{
    lv_sim *s0 = b->sims[0];
    cudaGraph_t gg = nullptr;
    LV_CUDA(s0, cudaGraphCreate(&gg, 0));
    cudaError_t e = cudaStreamBeginCaptureToGraph(s0->stream, gg, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed);
    if (e != cudaSuccess) { cudaGraphDestroy(gg); return cuda_fail(s0, e, "cudaStreamBeginCaptureToGraph"); }
    int rc = LV_OK;
    e = cudaEventRecord(b->ev[0], s0->stream);
    for (int r = 1; r < b->n && e == cudaSuccess; ++r) e = cudaStreamWaitEvent(b->sims[r]->stream, b->ev[0], 0);
    for (int r = 0; r < b->n && e == cudaSuccess && rc == LV_OK; ++r) {
        lv_sim *s = b->sims[r];
        for (int k = 0; k < steps && rc == LV_OK; ++k) {
            if (s->list_cap != 0) {          // list step: its own IF node around the rebuild chain
                rc = enqueue_list_step_if(s, gg, nullptr);
            } else {
                s->hashed = s->sort_mode == LV_SORT_COUNTING;     // steady-state step
                rc = enqueue_step(s);
            }
        }
        s->hashed = false;
        if (r > 0 && rc == LV_OK) {
            e = cudaEventRecord(b->ev[r], s->stream);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(s0->stream, b->ev[r], 0);
        }
    }
    cudaGraph_t gout = nullptr;
    cudaError_t e2 = cudaStreamEndCapture(s0->stream, &gout);
    (void)cudaGetLastError();
    if (rc == LV_OK && e != cudaSuccess) rc = cuda_fail(s0, e, "lv_batch capture");
    if (rc == LV_OK && e2 != cudaSuccess) rc = cuda_fail(s0, e2, "cudaStreamEndCapture");
    if (rc == LV_OK) {
        e2 = cudaGraphInstantiate(x, gg, 0);
        if (e2 != cudaSuccess) rc = cuda_fail(s0, e2, "cudaGraphInstantiate");
    }
    if (rc != LV_OK) { cudaGraphDestroy(gg); return rc; }
    *g = gg;
    return LV_OK;
}
}  // namespace

extern "C" {

int lv_batch_destroy(lv_batch *b)
{
    if (!b) return LV_OK;
    if (b->sims && b->n > 0 && b->sims[0]) cudaStreamSynchronize(b->sims[0]->stream);
    if (b->exec1) cudaGraphExecDestroy(b->exec1);
    if (b->execk) cudaGraphExecDestroy(b->execk);
    if (b->graph1) cudaGraphDestroy(b->graph1);
    if (b->graphk) cudaGraphDestroy(b->graphk);
    if (b->ev) {
        for (int r = 0; r < b->n; ++r) if (b->ev[r]) cudaEventDestroy(b->ev[r]);
        free(b->ev);
    }
    free(b->sims);
    delete b;
    return LV_OK;
}

int lv_batch_create(lv_batch **out, lv_sim **sims, int n_sims, int steps_per_launch)
{
    if (!out || !sims || n_sims < 1 || n_sims > 4096 || steps_per_launch < 1 || steps_per_launch > 256) return LV_E_ARG;
    for (int r = 0; r < n_sims; ++r) {
        if (!sims[r]) return LV_E_ARG;
        if (!sims[r]->bound || !sims[r]->state_set) return LV_E_ORDER;
        if (sims[r]->stream == nullptr || sims[r]->n == 0 || sims[r]->tim_cap > 0) return LV_E_ARG;
        for (int q = 0; q < r; ++q) if (sims[q] == sims[r]) return LV_E_ARG;
    }
    lv_batch *b = new (std::nothrow) lv_batch();
    if (!b) return LV_E_NOMEM;
    b->n = n_sims;
    b->chunk = steps_per_launch;
    b->sims = (lv_sim **)malloc(sizeof(lv_sim *) * n_sims);
    b->ev = (cudaEvent_t *)calloc(n_sims, sizeof(cudaEvent_t));
    if (!b->sims || !b->ev) { lv_batch_destroy(b); return LV_E_NOMEM; }
    memcpy(b->sims, sims, sizeof(lv_sim *) * n_sims);
    for (int r = 0; r < n_sims; ++r)
        if (cudaEventCreateWithFlags(&b->ev[r], cudaEventDisableTiming) != cudaSuccess) { lv_batch_destroy(b); return LV_E_CUDA; }
    int rc = capture_batch(b, 1, &b->graph1, &b->exec1);
    if (rc == LV_OK && b->chunk > 1) rc = capture_batch(b, b->chunk, &b->graphk, &b->execk);
    if (rc != LV_OK) { lv_batch_destroy(b); return rc; }
    *out = b;
    return LV_OK;
}

int lv_batch_step(lv_batch *b, int n)
{
    if (!b || n < 0) return LV_E_ARG;
    if (n == 0) return LV_OK;
    lv_sim *s0 = b->sims[0];
    // everything enqueued on the replicas' own streams so far comes first
    for (int r = 1; r < b->n; ++r) {
        LV_CUDA(s0, cudaEventRecord(b->ev[r], b->sims[r]->stream));
        LV_CUDA(s0, cudaStreamWaitEvent(s0->stream, b->ev[r], 0));
    }
    for (int r = 0; r < b->n; ++r) {
        lv_sim *s = b->sims[r];
        if (s->sort_mode == LV_SORT_COUNTING && s->list_cap == 0 && !s->hashed) {
            LV_CUDA(s0, lvk_hash_count(s->dev, s->bufs, false, s0->stream));     // the graph is the steady-state step
            s->hashed = true;
        }
        s->force_order_b = false;
    }
    int left = n;
    while (left > 0) {
        if (b->execk && left >= b->chunk) { LV_CUDA(s0, cudaGraphLaunch(b->execk, s0->stream)); left -= b->chunk; }
        else { LV_CUDA(s0, cudaGraphLaunch(b->exec1, s0->stream)); left -= 1; }
    }
    // ... and the replicas' own streams see the result
    LV_CUDA(s0, cudaEventRecord(b->ev[0], s0->stream));
    for (int r = 1; r < b->n; ++r) LV_CUDA(s0, cudaStreamWaitEvent(b->sims[r]->stream, b->ev[0], 0));
    return LV_OK;
}

}  // extern "C"

// ---- one entry point that allocates nothing and needs no caller scratch ------------------
// lv_observe_rdf_noalloc: the RDF pair walk (k_rdf_hist) with its histogram scratch in a
// file-scope device array instead of the caller's workspace.  The array's name is a host-side
// stand-in in host code: its device address is taken once per device, with that device current,
// by cudaGetSymbolAddress, and THAT pointer goes to the kernel.  Every GPU that loads the
// library holds the array (LV_NOALLOC_MAX_BINS * 8 bytes = 32 KiB) until the process exits.
static __device__ __align__(256) unsigned long long g_rdf_scratch[LV_NOALLOC_MAX_BINS];

namespace {
constexpr int kMaxDevices = 64;
unsigned long long *g_rdf_scratch_ptr[kMaxDevices];     // device address per device; nullptr: not taken yet

// device address of g_rdf_scratch on the CURRENT device
int rdf_scratch_of_current_device(lv_sim *s, unsigned long long **out)
{
    int dev = -1;
    LV_CUDA(s, cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return LV_E_ARG;
    if (!g_rdf_scratch_ptr[dev]) {
        unsigned long long *p = nullptr;
        LV_CUDA(s, cudaGetSymbolAddress((void **)&p, g_rdf_scratch));
        if (!p) return LV_E_CUDA;
        g_rdf_scratch_ptr[dev] = p;      // (two threads racing here store the same address)
    }
    *out = g_rdf_scratch_ptr[dev];
    return LV_OK;
}
}  // namespace

extern "C" int lv_observe_rdf_noalloc(lv_sim *s, double dr, int n_bins, uint64_t *hist, double *g)
{
    if (!s || !(dr > 0.0) || n_bins < 1) return LV_E_ARG;
    if (n_bins > LV_NOALLOC_MAX_BINS) {
        fprintf(stderr, "lv_observe_rdf_noalloc: n_bins = %d exceeds LV_NOALLOC_MAX_BINS = %d "
                        "(the static scratch array); use lv_observe_rdf\n", n_bins, LV_NOALLOC_MAX_BINS);
        return LV_E_CAPACITY;
    }
    if (!s->bound || !s->state_set) return LV_E_ORDER;
    if (hist) memset(hist, 0, 8 * (size_t)n_bins);
    if (g) for (int k = 0; k < n_bins; ++k) g[k] = 0.0;
    for (int b = 0; b < s->n_types; ++b)       // the pair walk keeps its stencil half-width in an int8
        if (std::ceil(dr * (double)n_bins * (1.0 + 1.0 / 1024.0) / s->grid.h[b]) > 100.0) return LV_E_ARG;
    if (s->n == 0) return LV_OK;
    unsigned long long *dh = nullptr;
    int rc = rdf_scratch_of_current_device(s, &dh);
    if (rc != LV_OK) return rc;
    // cell structures of the current state (steps (i) of PAPER.md:64), then the pair walk
    for (int k = 0; k < 3; ++k) {
        rc = enqueue_stage(s, k);
        if (rc != LV_OK) return rc;
    }
    // the array keeps the last call's counts: the kernel adds, so it must start at zero
    LV_CUDA(s, cudaMemsetAsync(dh, 0, 8 * (size_t)n_bins, s->stream));
    LV_CUDA(s, lvk_rdf_hist(s->dev, s->bufs, s->grid.h, dr, n_bins, dh, s->stream));
    uint64_t stack_hist[LV_NOALLOC_MAX_BINS];                      // 32 KiB of host stack, no heap either
    uint64_t *hh = hist ? hist : stack_hist;
    LV_CUDA(s, cudaMemcpyAsync(hh, dh, 8 * (size_t)n_bins, cudaMemcpyDeviceToHost, s->stream));
    LV_CUDA(s, cudaStreamSynchronize(s->stream));
    LvDevState st;
    LV_CUDA(s, cudaMemcpy(&st, s->bufs.st, sizeof(st), cudaMemcpyDeviceToHost));
    // Eq. 6: g_k = (psi_k / N) / ((N - 1) dV_k / V), V the droplet volume at this step
    const double R = lv_radius_of(s->sched_mode, s->R0, s->R1, s->sched_steps, st.step);
    const double V = 4.0 / 3.0 * M_PI * R * R * R, N = (double)s->n;
    if (g && s->n > 1)
        for (int k = 0; k < n_bins; ++k) g[k] = ((double)hh[k] / N) / ((N - 1.0) * shell_volume(k, dr) / V);
    return LV_OK;
}

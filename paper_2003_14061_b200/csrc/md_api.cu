// C-ABI layer of the MD hot path: argument checks, device memory, the time-step driver.  All arithmetic
// of the method runs in the kernels of md_kernels.cu; the host loop below only enqueues them (PAPER.md:79:
// "Essentially all computation is done on the GPU").  See include/md_b200.h for the contract of each call.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "md_init.h"
#include "md_types.h"

namespace {

thread_local char g_err[512] = "";

void set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

md_alloc_fn g_alloc = nullptr;
md_free_fn g_free = nullptr;
void *g_alloc_user = nullptr;

#define CK(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e__ = (call);                                                                  \
        if (e__ != cudaSuccess) {                                                                  \
            set_error("%s failed at %s:%d: %s", #call, __FILE__, __LINE__, cudaGetErrorString(e__)); \
            return MD_ERR_CUDA;                                                                    \
        }                                                                                          \
    } while (0)

struct EvPair {
    cudaEvent_t a, b;
    int cls;
};

}  // namespace

struct md_system {
    md_params prm;
    MdDev P;
    MdLaunch lc;
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    int device = 0;
    int sm_count = 0;
    char device_name[64] = "";
    std::vector<void *> allocs;
    md_alloc_fn alloc = nullptr;   // the hooks in force when the system was created: its memory goes back the way it came
    md_free_fn free_ = nullptr;
    void *alloc_user = nullptr;
    int64_t bytes = 0;
    DevCtrl *h_ctrl = nullptr;     // pinned, mapped
    DevCtrl *d_h_ctrl = nullptr;   // the device's address of h_ctrl
    double *h_stage = nullptr;     // pinned staging, 6 N doubles
    // double-buffered host I/O (md_stage_state / md_commit_state / md_get_state_async): copy streams and staging buffers
    cudaStream_t up_stream = nullptr, down_stream = nullptr;
    cudaEvent_t ev_up[2] = {nullptr, nullptr}, ev_exported = nullptr, ev_down[4] = {nullptr, nullptr, nullptr, nullptr};
    double *io_in[2] = {nullptr, nullptr}, *io_out[2] = {nullptr, nullptr};    // device, 6 N doubles each (xyz | vxyz, original order), on first use
    int in_head = 0, n_staged = 0;   // FIFO of staged states: slots in_head, in_head + 1 (mod 2)
    int64_t n_down = 0;              // downloads started; download d: staging buffer d % 2, event d % 4
    int64_t step = 0;
    int64_t launches = 0;
    bool has_state = false;
    bool stepped = false;
    int n_bonds_max = 0;
    double r_n = 0, cell_w = 0;
    // profiling
    bool profiling = false;
    std::vector<EvPair> pending, pool;
    // CUDA graph of one fused step: force+kick+drift -> decide -> IF(need_rebuild){cells, reorder, build}
    cudaGraph_t graph[3] = {nullptr, nullptr, nullptr};    // [0] kick+drift step head, [1] one fused force+kick+drift step, [2] GRAPH_UNROLL of them
    cudaGraphExec_t gexec[3] = {nullptr, nullptr, nullptr};
    cudaStream_t cap_stream = nullptr;
    bool graph_tried = false;
    int chain_kernels = 0;         // kernels inside the conditional body
    bool persist = false;          // small system: md_step runs as one cooperative launch
    int rebuilds_seen = 0;
    int64_t graph_steps = 0;       // steps run through the graph since the last status read         // ctrl->n_rebuilds at the last status read (launch accounting)
    double t_ms[MD_T_COUNT] = {0};
    int64_t t_n[MD_T_COUNT] = {0};
};

namespace {

void *dev_alloc(md_system *s, size_t bytes)
{
    void *p = nullptr;
    bytes = (bytes + 255) & ~(size_t)255;
    if (s->alloc) p = s->alloc(bytes, (void *)s->stream, s->alloc_user);
    else if (cudaMalloc(&p, bytes) != cudaSuccess) p = nullptr;
    if (!p) return nullptr;
    s->allocs.push_back(p);
    s->bytes += (int64_t)bytes;
    cudaMemsetAsync(p, 0, bytes, s->stream);
    return p;
}

void dev_free_all(md_system *s)
{
    for (void *p : s->allocs) {
        if (s->alloc) { if (s->free_) s->free_(p, s->alloc_user); }
        else cudaFree(p);
    }
    s->allocs.clear();
}

// RAII bracket: CUDA events around one launch wrapper while profiling is on
struct Timed {
    md_system *s;
    EvPair ev;
    bool on;
    Timed(md_system *s_, int cls, int n_launch) : s(s_), on(s_->profiling)
    {
        s->launches += n_launch;
        s->t_n[cls] += n_launch;
        if (!on) return;
        if (!s->pool.empty()) { ev = s->pool.back(); s->pool.pop_back(); }
        else { cudaEventCreate(&ev.a); cudaEventCreate(&ev.b); }
        ev.cls = cls;
        cudaEventRecord(ev.a, s->stream);
    }
    ~Timed()
    {
        if (!on) return;
        cudaEventRecord(ev.b, s->stream);
        s->pending.push_back(ev);
    }
};

void resolve_timers(md_system *s)
{
    for (EvPair &e : s->pending) {
        cudaEventSynchronize(e.b);
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, e.a, e.b) == cudaSuccess) s->t_ms[e.cls] += (double)ms;
        s->pool.push_back(e);
    }
    s->pending.clear();
}

int fetch_ctrl(md_system *s)
{
    mdk_publish_ctrl(s->P, s->d_h_ctrl, s->stream);          // a kernel, not a copy: see k_publish_ctrl
    s->launches += 1;
    CK(cudaStreamSynchronize(s->stream));
    CK(cudaGetLastError());
    return MD_OK;
}

int check_device_status(md_system *s)
{
    int rc = fetch_ctrl(s);
    if (rc) return rc;
    if (s->graph_steps > 0) {      // kernels of the conditional bodies that actually ran
        const int d = s->h_ctrl->n_rebuilds - s->rebuilds_seen;
        if (d > 0) s->launches += (int64_t)std::min<int64_t>(d, s->graph_steps) * s->chain_kernels;
        s->graph_steps = 0;
    }
    s->rebuilds_seen = s->h_ctrl->n_rebuilds;
    const int err = s->h_ctrl->err;
    if (err) {
        switch (err) {
        case MD_ERR_NEBR_OVERFLOW:
            set_error("neighbor matrix overflow: some atom has more than Mmax = %d neighbors", s->P.Mmax);
            break;
        case MD_ERR_BOND_BROKEN: set_error("FENE bond stretched to r >= R0"); break;
        case MD_ERR_NONFINITE: set_error("non-finite position or velocity"); break;
        case MD_ERR_CELL_OVERFLOW:
            set_error("MD_FLAG_LAYER_H: a cell holds more than N_l = %d atoms", s->P.n_layers);
            break;
        case MD_ERR_TILE_OVERFLOW:
            set_error("tiled W: a block's cell neighbourhood holds more than %d atoms; re-create with MD_FLAG_GLOBAL_W", s->P.tg.cap);
            break;
        default: set_error("device error %d", err);
        }
    }
    return err;
}

// cells + reorder + neighbor matrix.  Always enqueued; the kernels return at once unless the device-side
// decision (decide() in md_kernels.cu) asked for a rebuild.
void enqueue_rebuild(md_system *s)
{
    { Timed t(s, MD_T_CELLS, mdk_launches_of(LK_CELLS)); mdk_cells(s->P, s->lc, s->stream); }
    { Timed t(s, MD_T_REORDER, (s->P.has_bonds ? 2 : 1) + (s->P.layer_H ? 1 : 0)); mdk_reorder(s->P, s->lc, s->stream); }
    { Timed t(s, MD_T_NEBR, s->P.layer_H ? 2 : 1); if (s->P.tile_build) mdk_tile_build(s->P, s->stream); else mdk_build(s->P, s->lc, s->stream); }
}

void enqueue_force(md_system *s, int mode)
{
    const MdDev &P = s->P;
    if (P.tiled) mdk_tile_force(P, mode, s->stream);
    else mdk_force(P, s->lc, mode, s->stream);
}

// rebuild decision after a drifting kernel; cond: conditional handle of the step graph or 0
void enqueue_decide(md_system *s, bool fused_force, unsigned long long cond = 0ull)
{
    Timed t(s, MD_T_DECIDE, 1);
    mdk_decide(s->P, fused_force, s->stream, cond);
}

void drop_graph(md_system *s)
{
    for (int k = 0; k < 3; k++) {
        if (s->gexec[k]) cudaGraphExecDestroy(s->gexec[k]);
        if (s->graph[k]) cudaGraphDestroy(s->graph[k]);
        s->gexec[k] = nullptr; s->graph[k] = nullptr;
    }
    s->graph_tried = false;
}

// The drifting part of a time step as a CUDA graph: kind 0 = opening half kick + drift (k_kick_drift), kind 1 =
// fused force + kick + drift (k_force<1> / k_tile_force<1>); then k_decide; then the rebuild chain in the body
// of an IF node whose condition k_decide sets on the device (cudaGraphSetConditional).  A step without a
// rebuild so launches 2 kernels instead of 2 + 7 that find need_rebuild == 0 (PAPER.md:64 takes this decision
// on the host every step).  Returns false (and leaves no graph) if any step of the construction is refused;
// md_step then launches the kernels one by one.
#ifndef MD_GRAPH_UNROLL
#define MD_GRAPH_UNROLL 8
#endif
constexpr int GRAPH_UNROLL = MD_GRAPH_UNROLL;     // fused steps per launch of graph[2]: amortises the per-launch cost of a graph (small systems);
                                                  // 16 and 32 measured: no further gain (per-step overhead 4.7 / 5.5 / 5.7 us at N = 2M)

bool build_step_graph(md_system *s, int kind)
{
    cudaStream_t st = s->stream;
    if (!s->cap_stream && cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); return false; }
    const int reps = kind == 2 ? GRAPH_UNROLL : 1;
    const bool fused = kind >= 1;
    // The rebuild decision is its own one-block kernel (k_decide).  Taking it in the last block of the drifting kernel
    // (the paper's "last block done"; one or two levels of block counters) was measured slower at every
    // grid size, 32 to 16,384 blocks (wca_4k 22.1 vs 20.1 us per step, wca_262k 44.6 vs 41.0, wca_2m 206 vs 194): its chain
    // of fences, atomics and dependent loads at the tail of the kernel is longer than the launch it saves.  DESIGN.md 6f.
    cudaGraph_t g = nullptr;
    bool capturing = false, ok = false;
    do {
        if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) != cudaSuccess) break;
        capturing = true;
        bool bad = false;
        for (int rep = 0; rep < reps && !bad; rep++) {
            bad = true;
            cudaStreamCaptureStatus status;
            const cudaGraphNode_t *deps = nullptr;
            size_t ndeps = 0;
            if (cudaStreamGetCaptureInfo(st, &status, nullptr, &g, &deps, &ndeps) != cudaSuccess || !g) break;
            cudaGraphConditionalHandle h;
            if (cudaGraphConditionalHandleCreate(&h, g, 0, cudaGraphCondAssignDefault) != cudaSuccess) break;
            if (fused) enqueue_force(s, 1);
            else mdk_kick_drift(s->P, s->lc, st);
            mdk_decide(s->P, fused, st, (unsigned long long)h);
            if (cudaStreamGetCaptureInfo(st, &status, nullptr, &g, &deps, &ndeps) != cudaSuccess) break;
            cudaGraphNodeParams cp = {cudaGraphNodeTypeConditional};
            cp.conditional.handle = h;
            cp.conditional.type = cudaGraphCondTypeIf;
            cp.conditional.size = 1;
            cudaGraphNode_t cnode;
            if (cudaGraphAddNode(&cnode, g, deps, ndeps, &cp) != cudaSuccess) break;
            cudaGraph_t body = cp.conditional.phGraph_out[0];
            if (cudaStreamBeginCaptureToGraph(s->cap_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal) != cudaSuccess) break;
            mdk_cells(s->P, s->lc, s->cap_stream);
            mdk_reorder(s->P, s->lc, s->cap_stream);
            if (s->P.tile_build) mdk_tile_build(s->P, s->cap_stream); else mdk_build(s->P, s->lc, s->cap_stream);
            cudaGraph_t body_out = nullptr;
            if (cudaStreamEndCapture(s->cap_stream, &body_out) != cudaSuccess) break;
            if (cudaStreamUpdateCaptureDependencies(st, &cnode, 1, cudaStreamSetCaptureDependencies) != cudaSuccess) break;
            bad = false;
        }
        if (bad) break;
        capturing = false;
        if (cudaStreamEndCapture(st, &g) != cudaSuccess) { g = nullptr; break; }
        s->graph[kind] = g;
        if (cudaGraphInstantiate(&s->gexec[kind], g, 0) != cudaSuccess) break;
        ok = true;
    } while (0);
    if (!ok) {
        if (capturing) { cudaGraph_t junk = nullptr; cudaStreamEndCapture(st, &junk); if (junk) cudaGraphDestroy(junk); }
        cudaGetLastError();
        if (s->gexec[kind]) { cudaGraphExecDestroy(s->gexec[kind]); s->gexec[kind] = nullptr; }
        if (s->graph[kind]) { cudaGraphDestroy(s->graph[kind]); s->graph[kind] = nullptr; }
        return false;
    }
    s->chain_kernels = mdk_launches_of(LK_CELLS) + (s->P.has_bonds ? 2 : 1) + 1 + (s->P.layer_H ? 2 : 0);
    return true;
}

// both graphs, once; all or nothing
bool have_graphs(md_system *s)
{
    if (s->profiling || (s->prm.flags & MD_FLAG_NO_GRAPH)) return false;
    if (!s->graph_tried) {
        s->graph_tried = true;
        const bool fused = s->prm.step_mode == MD_STEP_FUSED;
        if (!build_step_graph(s, 0) || (fused && (!build_step_graph(s, 1) || !build_step_graph(s, 2)))) {
            const bool tried = true;
            drop_graph(s);
            s->graph_tried = tried;
        }
    }
    return s->gexec[0] != nullptr;
}

void enqueue_forces_only(md_system *s)
{
    if (s->P.half_list) { Timed t(s, MD_T_FORCE, 2); mdk_force_newton3(s->P, s->lc, s->stream); }
    else { Timed t(s, MD_T_FORCE, 1); enqueue_force(s, 0); }
}

// state already in scratch (xyz | vxyz, original order): load, bin, build W, evaluate forces
int install_state(md_system *s)
{
    s->launches += 2;
    mdk_load_state(s->P, s->stream);
    mdk_force_rebuild(s->P, s->stream);
    enqueue_rebuild(s);
    enqueue_forces_only(s);
    s->step = 0;
    s->stepped = false;
    s->has_state = true;
    int rc = check_device_status(s);
    if (rc) return rc;
    // the initial build is not counted as a rebuild
    s->h_ctrl->n_rebuilds = 0;
    s->rebuilds_seen = 0;
    CK(cudaMemsetAsync(&s->P.ctrl->n_rebuilds, 0, sizeof(int), s->stream));
    return MD_OK;
}

// page-locked host memory can be the source / target of the asynchronous copies directly; anything else goes
// through the library's pinned staging buffer
bool is_pinned(const void *p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeHost;
}

// check: validate the coordinate range on the device (md_set_state) before anything of the old state is touched
int upload_state(md_system *s, const double *xyz, const double *vxyz, bool check = false)
{
    const size_t n3 = 3 * (size_t)s->P.N;
    if (!vxyz) {   // keep velocities: bring them to original order in the second half of scratch first
        if (!s->has_state) { set_error("md_set_state: no velocities to keep"); return MD_ERR_INVALID; }
        s->launches += 1;
        mdk_export(s->P, 1, s->P.scratch + n3, s->stream);
    }
    const double *src = xyz;
    if (!is_pinned(xyz)) { memcpy(s->h_stage, xyz, n3 * sizeof(double)); src = s->h_stage; }
    CK(cudaMemcpyAsync(s->P.scratch, src, n3 * sizeof(double), cudaMemcpyHostToDevice, s->stream));
    if (vxyz) {
        src = vxyz;
        if (!is_pinned(vxyz)) { memcpy(s->h_stage + n3, vxyz, n3 * sizeof(double)); src = s->h_stage + n3; }
        CK(cudaMemcpyAsync(s->P.scratch + n3, src, n3 * sizeof(double), cudaMemcpyHostToDevice, s->stream));
    }
    if (check) {
        s->launches += 1;
        mdk_check_range(s->P, s->prm.box, s->stream);
        int rc = fetch_ctrl(s);
        if (rc) return rc;
        if (s->h_ctrl->err == MD_ERR_INVALID) {
            CK(cudaMemsetAsync(&s->P.ctrl->err, 0, sizeof(int), s->stream));
            const double L = s->prm.box;
            for (size_t i = 0; i < n3; i++)
                if (!(xyz[i] >= 0.0 && xyz[i] <= L)) { set_error("md_set_state: coordinate %zu = %g outside [0, L]", i, xyz[i]); break; }
            return MD_ERR_INVALID;
        }
    }
    return install_state(s);
}

int download(md_system *s, int what, double *out)
{
    if (!s || !out) { set_error("null argument"); return MD_ERR_INVALID; }
    if (!s->has_state) { set_error("no state loaded"); return MD_ERR_INVALID; }
    const size_t n3 = 3 * (size_t)s->P.N;
    s->launches += 1;
    mdk_export(s->P, what, s->P.scratch, s->stream);
    const bool direct = is_pinned(out);
    CK(cudaMemcpyAsync(direct ? out : s->h_stage, s->P.scratch, n3 * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    CK(cudaGetLastError());
    if (!direct) memcpy(out, s->h_stage, n3 * sizeof(double));
    return MD_OK;
}

// positions / velocities / forces in original-id order into a caller-owned DEVICE buffer: one kernel, no copy, no sync
int export_device(md_system *s, int what, double *dst)
{
    if (!s || !dst) { set_error("null argument"); return MD_ERR_INVALID; }
    if (!s->has_state) { set_error("no state loaded"); return MD_ERR_INVALID; }
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, dst) != cudaSuccess || (a.type != cudaMemoryTypeDevice && a.type != cudaMemoryTypeManaged)) {
        cudaGetLastError();
        set_error("the *_device getters need a device pointer");
        return MD_ERR_INVALID;
    }
    s->launches += 1;
    mdk_export(s->P, what, dst, s->stream);
    CK(cudaGetLastError());
    return MD_OK;
}

// Box of cells per thread block, block size and tile capacity of the tiled W layout (md_types.h: TileGeom).
// Defaults aim at ~0.8 own atoms per thread and a 2 x 2 cross-section in y, z (halo factor ~4.5 for the WCA
// configs); md_params.tile_cells / tile_threads / tile_capacity override them (tuning runs, box-shape tests).
bool choose_tile(MdDev &P, const md_params &prm, size_t smem_optin, bool for_tiled_w)
{
    TileGeom &G = P.tg;
    const int nc = P.nc;
    const double per_cell = (double)P.N1 / ((double)nc * nc * nc);      // atoms per r_n-wide cell
    auto knob = [](int v, int dflt) { return v > 0 ? v : dflt; };
    // Build for the global-index W of short-column systems (a few atoms per cell): boxes of S x 3 x 3 cells -- a third less halo
    // to stage per own atom than S x 2 x 2 -- for 256-thread blocks filled to <= 92 %.  Measured, build per
    // rebuild: wca_2m_dr03 0.338 -> 0.303 ms (11 x 3 x 3 against 20 x 2 x 2 @ 224 threads), dr05 0.376 -> 0.349, chains_1m 0.193 -> 0.177.
    const bool short_cols = !for_tiled_w && per_cell <= 8.0;
    G.R = std::min(std::max(knob(prm.tile_cells[1], short_cols ? 3 : 2), 1), 3);
    G.RZ = std::min(std::max(knob(prm.tile_cells[2], short_cols ? 3 : 2), 1), 3);
    G.threads = knob(prm.tile_threads, per_cell > 8.0 ? 512 : 256);
    if (G.threads < 64 || G.threads > 512 || G.threads % 32) { set_error("tile_threads must be a multiple of 32 in [64, 512]"); return false; }
    // box length along x in r_n-wide cells; in fine cells it is a multiple of kx, so every box starts at least kx cells
    // from the row's ends or exactly at them: the halo of a box is then one contiguous range on either side (md_types.h)
    int S = prm.tile_cells[0];
    if (S <= 0 && for_tiled_w && prm.tile_threads <= 0) {
        // Tiled force kernel (long columns): blocks of 256 threads filled to <= 92 % with own atoms -- four resident blocks
        // per SM overlap one block's staging with the others' columns, and a box that owns more atoms than the block has
        // threads costs a second pass.  Measured: lj_1m 3 x 2 x 2 cells @ 256 threads 3.54 G against
        // 5 x 2 x 2 @ 512 (the round-1 rule) 3.32 G; the paper's LJ state point 5 x 2 x 2 @ 256 4.88 G against 9 x 2 x 2 @ 512 4.40 G.
        const double q = G.R * G.RZ * per_cell;                        // own atoms per cell of box length
        const int s256 = std::max(1, (int)floor(0.92 * 256 / q)), s512 = std::max(1, (int)floor(0.92 * 512 / q));
        const double f256 = s256 * q / 256.0, f512 = s512 * q / 512.0;
        const bool small = f256 <= 1.0 && (f256 >= 0.75 || f256 >= f512 || f512 > 1.0);
        G.threads = small ? 256 : 512;
        S = small ? s256 : s512;
    }
    if (S <= 0 && short_cols && prm.tile_threads <= 0) S = std::max(1, (int)floor(0.92 * G.threads / (G.R * G.RZ * per_cell)));
    if (S <= 0) S = (int)lround(0.8 * G.threads / (G.R * G.RZ * per_cell));
    S = std::min(std::max(S, 1), nc);
    G.nsx = (nc + S - 1) / S;
    S = (nc + G.nsx - 1) / G.nsx;                   // balance the boxes along x
    G.nsx = (nc + S - 1) / S;
    if (prm.tile_threads <= 0) {
        // small boxes (few cells per edge): S was clipped to the row, so shrink the block to the atoms a box owns
        const double own = (double)S * G.R * G.RZ * per_cell;
        int t = 32 * (int)ceil(1.12 * own / 32.0);
        if (for_tiled_w) t = t <= 128 ? 128 : (t <= 256 ? 256 : 512);      // instantiated sizes of the tiled force kernels
        G.threads = std::min(G.threads, std::max(64, t));
    }
    G.S = S * P.kx;
    G.nsy = (nc + G.R - 1) / G.R;
    G.nsz = (nc + G.RZ - 1) / G.RZ;
    G.nsys = P.n_sys;
    const double mean = (double)(S + 2) * (G.R + 2) * (G.RZ + 2) * per_cell;
    int cap = prm.tile_capacity;
    if (cap <= 0) cap = (int)((for_tiled_w ? 1.25 : 1.35) * mean + 6.0 * sqrt(mean) + 32.0);     // tiled force: four 54 KB tiles per SM at lj_1m
    cap = (cap + 31) & ~31;
    if (cap > 8192) cap = 8192;
    G.cap = cap;
    // the largest tile the build kernel's shared memory holds (positions + cell table + index table for global-index W)
    P.tiled = for_tiled_w ? 1 : 0;                  // mdk_tile_smem depends on the W layout
    while (G.cap > 64 && mdk_tile_smem(P, true) + 8192 > smem_optin) G.cap -= 32;
    cap = G.cap;
    if (mean > 0.8 * cap) { set_error("tile build: %.0f atoms per tile exceed the tile capacity %d; use MD_FLAG_GLOBAL_W or a smaller tile_cells[0]", mean, cap); return false; }
    if (mdk_tile_smem(P, true) + 8192 > smem_optin) { set_error("tile build: tile of %d atoms does not fit shared memory", cap); return false; }
    return true;
}

}  // namespace

void mdk_set_error(const char *msg) { set_error("%s", msg); }

extern "C" {

const char *md_last_error(void) { return g_err; }
const char *md_version(void) { return "md_b200 0.1 (sm_100a)"; }

void md_set_allocator(md_alloc_fn alloc, md_free_fn free_, void *user)
{
    g_alloc = alloc;
    g_free = free_;
    g_alloc_user = user;
}

void md_params_default(md_params *p)
{
    if (!p) return;
    memset(p, 0, sizeof(*p));
    p->temperature = 1.0;
    p->lattice = MD_LATTICE_AUTO;
    p->force_variant = MD_FORCE_FULL_LIST;
    p->step_mode = MD_STEP_FUSED;
    p->device = -1;
}

void md_destroy(md_system *s)
{
    if (!s) return;
    if (s->stream) cudaStreamSynchronize(s->stream);
    for (cudaStream_t t : {s->up_stream, s->down_stream}) if (t) { cudaStreamSynchronize(t); cudaStreamDestroy(t); }
    for (cudaEvent_t e : {s->ev_up[0], s->ev_up[1], s->ev_exported, s->ev_down[0], s->ev_down[1], s->ev_down[2], s->ev_down[3]}) if (e) cudaEventDestroy(e);
    for (EvPair &e : s->pending) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
    for (EvPair &e : s->pool) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
    drop_graph(s);
    if (s->cap_stream) cudaStreamDestroy(s->cap_stream);
    dev_free_all(s);
    if (s->h_ctrl) cudaFreeHost(s->h_ctrl);
    if (s->h_stage) cudaFreeHost(s->h_stage);
    if (s->own_stream && s->stream) cudaStreamDestroy(s->stream);
    delete s;
}

md_system *md_create_ex(const md_params *pp)
{
    if (!pp) { set_error("md_create_ex: null params"); return nullptr; }
    md_params p = *pp;
    if (p.n_systems <= 0) p.n_systems = 1;
    if (p.n_atoms <= 0 || p.n_atoms * p.n_systems >= (1ll << 29)) { set_error("n_atoms * n_systems must be in [1, 2^29)"); return nullptr; }
    if (!(p.r_cut > 0) || !(p.r_shell >= 0) || !(p.dt > 0) || !(p.temperature >= 0)) {
        set_error("r_cut, dt must be > 0; r_shell, temperature >= 0");
        return nullptr;
    }
    if (p.box > 0) {
        if (p.density > 0) {
            const double d = (double)p.n_atoms / (p.box * p.box * p.box);
            if (fabs(d - p.density) > 1e-12 * p.density) { set_error("box and density disagree"); return nullptr; }
        }
    } else if (p.density > 0) {
        p.box = cbrt((double)p.n_atoms / p.density);
    } else {
        set_error("give box or density");
        return nullptr;
    }
    p.density = (double)p.n_atoms / (p.box * p.box * p.box);
    if (p.force_variant != MD_FORCE_FULL_LIST && p.force_variant != MD_FORCE_NEWTON3_ATOMICS) { set_error("bad force_variant"); return nullptr; }
    if (p.force_variant == MD_FORCE_NEWTON3_ATOMICS) p.step_mode = MD_STEP_SPLIT;
    if (p.step_mode != MD_STEP_FUSED && p.step_mode != MD_STEP_SPLIT) { set_error("bad step_mode"); return nullptr; }
    if (p.block_size == 0) p.block_size = 128;     // measured best by a small margin (the paper: 3 % spread)
    if (p.block_size != 64 && p.block_size != 128 && p.block_size != 256 && p.block_size != 512) {
        set_error("block_size must be 64, 128, 256 or 512");
        return nullptr;
    }
    if (p.precision != MD_PREC_F64 && p.precision != MD_PREC_F32) { set_error("bad precision"); return nullptr; }
    const bool sp = p.precision == MD_PREC_F32;
    if (sp && p.force_variant != MD_FORCE_FULL_LIST) { set_error("MD_PREC_F32 supports the full-list force variant only"); return nullptr; }
    if (sp && (p.flags & MD_FLAG_TILED_W)) { set_error("MD_PREC_F32 uses the global-index W layout"); return nullptr; }
    if (p.flags & MD_FLAG_LAYER_H) {
        if (sp || p.force_variant != MD_FORCE_FULL_LIST || p.n_systems > 1 || (p.flags & MD_FLAG_TILED_W)) {
            set_error("MD_FLAG_LAYER_H: fp64, full-list variant, one system, global-index W only");
            return nullptr;
        }
        p.flags |= MD_FLAG_GLOBAL_W;
    } else {
        p.reorder_interval = 0;
    }
    const double rn = p.r_cut + p.r_shell;
    // single precision: the box edge is the binary32 number, and cells keep a margin above the rounding error of a
    // binary32 r^2 (~2e-7 relative) so that no accepted pair can lie outside the 27-cell stencil
    const double box_eff = sp ? (double)(float)p.box : p.box;
    int nc = (int)floor(box_eff / rn);
    if (nc >= 1 && box_eff / nc - rn < (sp ? 1e-5 : 1e-9) * rn) nc -= 1;     // keep the cell strictly wider than r_n
    if (nc < 3) { set_error("box too small: %d cells per edge (need >= 3)", nc); return nullptr; }
    if (p.cell_split_x < 0 || p.cell_split_x > 8) { set_error("cell_split_x must be in [0, 8]"); return nullptr; }
    if (p.cell_split_x == 0) p.cell_split_x = (p.flags & MD_FLAG_LAYER_H) ? 1 : 2;      // measured: BASELINE.md sec. 4
    if ((p.flags & MD_FLAG_LAYER_H) && p.cell_split_x != 1) { set_error("MD_FLAG_LAYER_H keeps the paper's cubic cells (cell_split_x = 1)"); return nullptr; }
    if ((int64_t)nc * nc * nc * p.cell_split_x * std::max(1, p.n_systems) > (1ll << 30)) { set_error("too many cells"); return nullptr; }
    if (p.max_neighbors <= 0) {
        const double ideal = 4.0 / 3.0 * 3.14159265358979323846 * rn * rn * rn * p.density;
        p.max_neighbors = 16 * (int)ceil((1.35 * ideal + 12.0) / 16.0);
    }
    p.max_neighbors = (p.max_neighbors + 3) & ~3;          // W rows are stored in pairs in the tiled layout, padded to fours in single precision
    if (p.lattice == MD_LATTICE_AUTO) {
        p.lattice = md_init_pick_lattice(p.n_atoms);
        if (!p.lattice) { set_error("n_atoms fits neither a simple-cubic nor an FCC lattice"); return nullptr; }
    }

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        set_error("no CUDA device: this library has no CPU fallback");
        cudaGetLastError();
        return nullptr;
    }
    md_system *s = new md_system();
    s->prm = p;
    s->alloc = g_alloc; s->free_ = g_free; s->alloc_user = g_alloc_user;
    auto fail = [&](const char *what) -> md_system * {
        if (what) set_error("%s: %s", what, cudaGetErrorString(cudaGetLastError()));
        md_destroy(s);
        return nullptr;
    };
    if (p.device >= 0 && cudaSetDevice(p.device) != cudaSuccess) return fail("cudaSetDevice");
    if (cudaGetDevice(&s->device) != cudaSuccess) return fail("cudaGetDevice");
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, s->device) != cudaSuccess) return fail("cudaGetDeviceProperties");
    snprintf(s->device_name, sizeof(s->device_name), "%.63s", prop.name);
    s->sm_count = prop.multiProcessorCount;
    if (prop.major < 10) { set_error("device %s is sm_%d%d; this library is built for sm_100a only", prop.name, prop.major, prop.minor); md_destroy(s); return nullptr; }
    if (p.stream) s->stream = (cudaStream_t)p.stream;
    else {
        if (cudaStreamCreateWithFlags(&s->stream, cudaStreamNonBlocking) != cudaSuccess) return fail("cudaStreamCreate");
        s->own_stream = true;
    }

    MdDev &P = s->P;
    memset(&P, 0, sizeof(P));
    P.sm_count = prop.multiProcessorCount;
    P.n_sys = p.n_systems;
    P.N1 = (int)p.n_atoms;
    P.N = P.N1 * P.n_sys;
    P.N_pad = (P.N + 127) & ~127;
    P.Mmax = p.max_neighbors;
    P.nc = nc;
    P.kx = p.cell_split_x;
    P.ncx = nc * P.kx;
    P.NC1 = P.ncx * nc * nc;
    P.NC = P.NC1 * P.n_sys;
    P.half_list = p.force_variant == MD_FORCE_NEWTON3_ATOMICS;
    P.scan_blocks = (P.NC + 2047) / 2048;
    P.L = box_eff; P.half_L = 0.5 * box_eff; P.inv_w = (double)nc / box_eff;
    P.inv_wx = (double)P.ncx / box_eff;
    // row pruning of the neighbor build: binary32 constants rounded to the safe side (md_device.cuh: row_halfwidth)
    P.w_f = (float)(box_eff / nc * (1.0 - 1e-5));
    P.inv_wx_f = (float)(P.inv_wx * (1.0 + 1e-5));
    P.rn2_prune = (float)(rn * rn * (1.0 + 1e-5));
    P.sp = sp ? 1 : 0;
    // padded columns pay once a column is long enough (measured: +14 % at 76 neighbors, -5 % at 12; md_sp.cu)
    P.sp_pad = sp && 4.0 / 3.0 * 3.14159265358979323846 * rn * rn * rn * p.density >= 32.0 ? 4 : 1;
    P.Lf = (float)p.box; P.half_Lf = 0.5f * P.Lf;
    P.rc2f = (float)(p.r_cut * p.r_cut); P.rn2f = (float)(rn * rn);
    P.dtf = (float)p.dt; P.hdtf = (float)(0.5 * p.dt);
    P.rc2 = p.r_cut * p.r_cut;
    P.rn2 = rn * rn;
    { const double sc = 1.0 / P.rc2, sc3 = sc * sc * sc; P.uc = 4.0 * sc3 * (sc3 - 1.0); P.ucf = (float)P.uc; }
    P.dt = p.dt; P.hdt = 0.5 * p.dt; P.thresh = 0.5 * p.r_shell;
    s->r_n = rn; s->cell_w = box_eff / nc;
    s->lc.block = p.block_size;
    s->lc.grid_atoms = (P.N + p.block_size - 1) / p.block_size;

    P.tiled = 0;
    P.tile_build = 0;
    if (!P.half_list && !(p.flags & MD_FLAG_GLOBAL_W)) {
        // shared-memory staged neighbor build (both W layouts); the tiled W layout only on request
        const double mbar_est = 4.0 / 3.0 * 3.14159265358979323846 * rn * rn * rn * p.density;
        // (single precision: the tile-staged BUILD only; its force kernel gathers float4 records)
        const bool want_tiled = !sp && ((p.flags & MD_FLAG_TILED_W) || (!(p.flags & MD_FLAG_GATHER_W) && mbar_est >= 32.0));
        const bool fits = choose_tile(P, p, prop.sharedMemPerBlockOptin, want_tiled);
        if (!fits && (p.flags & MD_FLAG_TILED_W)) { md_destroy(s); return nullptr; }
        P.tile_build = fits ? 1 : 0;
        // the tile build addresses W with 32-bit element offsets (md_tile.cu: Emit); larger matrices use the gather build
        if ((uint64_t)p.max_neighbors * (uint64_t)((P.N + 127) & ~127) >= (1ull << 31)) P.tile_build = 0;
        // single precision, many small systems whose x-rows are shorter than the box length the tile wants: the gather
        // build is faster there (measured 64 / 512 x wca_4k: 6.90 vs 6.67 G and 13.75 vs 12.86 G atom-steps/s)
        if (sp && fits && P.n_sys >= 32 && P.tg.S >= P.ncx) P.tile_build = 0;
        // W layout: measured on B200, tile-local W wins once a column of W is long enough
        // to amortise staging the tile (LJ r_c = 2.5: 76 neighbors, +17 %) and loses for the short WCA columns
        // (12 neighbors, -17 %).  Estimated mean column length = ideal-gas count in the neighbor sphere.
        P.tiled = fits && P.tile_build && want_tiled ? 1 : 0;
        if (fits && mdk_tile_configure(P) != 0) {
            set_error("tile kernels: %d threads per block not available for this W layout, or cudaFuncSetAttribute failed", P.tg.threads);
            md_destroy(s);
            return nullptr;
        }
    } else if (p.flags & MD_FLAG_TILED_W) {
        set_error("MD_FLAG_TILED_W needs the full-list force variant and excludes MD_FLAG_GLOBAL_W");
        md_destroy(s);
        return nullptr;
    }
    if (p.flags & MD_FLAG_LAYER_H) {
        // N_l: the paper sizes H by the measured maximum occupancy (N3); here a fixed bound from the mean
        const double mean_occ = (double)P.N1 / P.NC1;
        P.layer_H = 1;
        P.n_layers = 8 * (int)ceil((2.0 * mean_occ + 8.0) / 8.0);
        P.reorder_interval = p.reorder_interval;
    }
    P.w_row = P.N_pad; P.w_col = 1;
    if (p.flags & MD_FLAG_W_TRANSPOSED) {
        if (P.tiled) { set_error("MD_FLAG_W_TRANSPOSED applies to the global-index W layout only"); md_destroy(s); return nullptr; }
        P.w_row = 1; P.w_col = P.Mmax;
    }
    // small systems run md_step as one cooperative launch (k_persist); it lists neighbors with the gathering build
    // -- the default for small systems only: any flag or tile setting that selects a path keeps the step graph
    const bool tile_knobs = pp->tile_cells[0] || pp->tile_cells[1] || pp->tile_cells[2] || pp->tile_threads || pp->tile_capacity;
    if (p.flags == 0 && !tile_knobs && p.step_mode == MD_STEP_FUSED && mdk_persist_ok(P)) {
        s->persist = true;
        P.tile_build = 0;
    }
    P.max_grid = std::max((P.N + 63) / 64, P.tile_build ? P.tg.nsx * P.tg.nsy * P.tg.nsz * P.tg.nsys : 0);

    const size_t np = (size_t)P.N_pad;
    bool ok = true;
    auto A = [&](size_t bytes) { void *q = dev_alloc(s, bytes); if (!q) ok = false; return q; };
    for (int k = 0; k < 2; k++) {
        if (sp) {
            P.posf[k] = (float4 *)A(np * sizeof(float4));
            P.velf[k] = (float4 *)A(np * sizeof(float4));
        } else {
            P.pos[k] = (pos_t *)A(np * sizeof(pos_t));
            P.vel[k] = (double *)A(3 * np * sizeof(double));
        }
        P.id[k] = (int *)A(np * sizeof(int));
    }
    if (sp) P.frcf = (float4 *)A(np * sizeof(float4));
    else P.frc = (double *)A(3 * np * sizeof(double));
    P.cell_of = (int *)A(np * sizeof(int));
    P.slot = (int *)A(np * sizeof(int));
    P.perm = (int *)A(np * sizeof(int));
    P.nnb = (int *)A(np * sizeof(int));
    P.cell_count = (int *)A(((size_t)P.NC + 1) * sizeof(int));
    P.cell_start = (int *)A(((size_t)P.NC + 1) * sizeof(int));
    P.block_sums = (int *)A(((size_t)P.scan_blocks + 1) * sizeof(int));
    P.W = (int *)A((size_t)(P.tiled ? P.Mmax / 2 : P.Mmax) * np * sizeof(int));
    if (P.layer_H) P.H = (int *)A((size_t)P.NC * P.n_layers * sizeof(int));
    P.partials = (double *)A((size_t)RED_N * P.max_grid * sizeof(double));
    P.blk_vmax2 = (double *)A(((size_t)P.max_grid + 64 + 2) * sizeof(double));     // 64 = DEC_SLOTS (md_device.cuh), then the persistent kernels' 2 x grid <= max_grid + 2
    if (P.tiled) P.tile_desc = (int *)A((size_t)P.tg.nsx * P.tg.nsy * P.tg.nsz * P.tg.nsys * sizeof(TileDesc));
    P.scratch = (double *)A(6 * (size_t)P.N * sizeof(double));
    P.ctrl = (DevCtrl *)A(sizeof(DevCtrl));
    if (!ok) { set_error("device allocation failed (%.1f MB so far)", s->bytes / 1048576.0); md_destroy(s); return nullptr; }
    if (cudaHostAlloc((void **)&s->h_ctrl, sizeof(DevCtrl), cudaHostAllocMapped) != cudaSuccess ||
        cudaHostGetDevicePointer((void **)&s->d_h_ctrl, s->h_ctrl, 0) != cudaSuccess) return fail("cudaHostAlloc (mapped)");
    if (cudaMallocHost((void **)&s->h_stage, 6 * (size_t)P.N * sizeof(double)) != cudaSuccess) return fail("cudaMallocHost");
    memset(s->h_ctrl, 0, sizeof(DevCtrl));

    if (p.lattice != MD_LATTICE_NONE) {
        std::vector<double> xyz(3 * (size_t)P.N), v(3 * (size_t)P.N);
        for (int b = 0; b < P.n_sys; b++) {      // every system: the same lattice, its own velocities (seed + b)
            const size_t o = 3 * (size_t)b * P.N1;
            if (!md_init_lattice(p.lattice, p.n_atoms, p.box, xyz.data() + o)) {
                set_error("n_atoms = %lld does not fit lattice %d", (long long)p.n_atoms, p.lattice);
                md_destroy(s);
                return nullptr;
            }
            md_init_velocities(p.n_atoms, p.temperature, p.seed + (uint64_t)b, v.data() + o);
        }
        if (upload_state(s, xyz.data(), v.data()) != MD_OK) { md_destroy(s); return nullptr; }
    } else if (cudaStreamSynchronize(s->stream) != cudaSuccess) {
        return fail("cudaStreamSynchronize");
    }
    return s;
}

md_system *md_create(int64_t n_atoms, double box, double density, double r_cut, double r_shell, double dt, uint64_t seed)
{
    md_params p;
    md_params_default(&p);
    p.n_atoms = n_atoms; p.box = box; p.density = density; p.r_cut = r_cut; p.r_shell = r_shell; p.dt = dt; p.seed = seed;
    return md_create_ex(&p);
}

int md_set_state(md_system *s, const double *xyz, const double *vxyz)
{
    if (!s || !xyz) { set_error("md_set_state: null argument"); return MD_ERR_INVALID; }
    if (s->P.rigid) { set_error("md_set_state: a rigid-molecule system takes its state through md_set_rigid_state"); return MD_ERR_INVALID; }
    return upload_state(s, xyz, vxyz, true);      // the range check [0, L] runs on the device, before the old state is touched
}

int md_set_state_device(md_system *s, const double *xyz_device, const double *vxyz_device)
{
    if (!s || !xyz_device) { set_error("md_set_state_device: null argument"); return MD_ERR_INVALID; }
    for (const double *p : {xyz_device, vxyz_device}) {
        cudaPointerAttributes a;
        if (p && (cudaPointerGetAttributes(&a, p) != cudaSuccess || (a.type != cudaMemoryTypeDevice && a.type != cudaMemoryTypeManaged))) {
            cudaGetLastError();
            set_error("md_set_state_device needs device pointers");
            return MD_ERR_INVALID;
        }
    }
    const size_t n3 = 3 * (size_t)s->P.N;
    if (!vxyz_device) {
        if (!s->has_state) { set_error("md_set_state_device: no velocities to keep"); return MD_ERR_INVALID; }
        s->launches += 1;
        mdk_export(s->P, 1, s->P.scratch + n3, s->stream);
    } else {
        CK(cudaMemcpyAsync(s->P.scratch + n3, vxyz_device, n3 * sizeof(double), cudaMemcpyDeviceToDevice, s->stream));
    }
    CK(cudaMemcpyAsync(s->P.scratch, xyz_device, n3 * sizeof(double), cudaMemcpyDeviceToDevice, s->stream));
    s->launches += 1;
    mdk_check_range(s->P, s->prm.box, s->stream);
    int rc = fetch_ctrl(s);
    if (rc) return rc;
    if (s->h_ctrl->err == MD_ERR_INVALID) {
        CK(cudaMemsetAsync(&s->P.ctrl->err, 0, sizeof(int), s->stream));
        set_error("md_set_state_device: a coordinate lies outside [0, L]");
        return MD_ERR_INVALID;
    }
    return install_state(s);
}

namespace {

// copy streams, events and the device staging buffers (two per direction) of the asynchronous I/O calls, on first use
int io_ready(md_system *s)
{
    if (s->P.rigid) { set_error("asynchronous state I/O: a rigid-molecule system exchanges its state through md_set/get_rigid_state"); return MD_ERR_INVALID; }
    if (s->up_stream) return MD_OK;
    const size_t bytes = 6 * (size_t)s->P.N * sizeof(double);
    for (int k = 0; k < 2; k++) {
        s->io_in[k] = (double *)dev_alloc(s, bytes);
        s->io_out[k] = (double *)dev_alloc(s, bytes);
        if (!s->io_in[k] || !s->io_out[k]) { set_error("asynchronous state I/O: out of device memory (4 x %zu bytes)", bytes); return MD_ERR_NOMEM; }
    }
    CK(cudaStreamSynchronize(s->stream));           // the buffers were cleared on the system's stream
    CK(cudaStreamCreateWithFlags(&s->up_stream, cudaStreamNonBlocking));
    CK(cudaStreamCreateWithFlags(&s->down_stream, cudaStreamNonBlocking));
    for (cudaEvent_t *e : {&s->ev_up[0], &s->ev_up[1], &s->ev_exported, &s->ev_down[0], &s->ev_down[1], &s->ev_down[2], &s->ev_down[3]})
        CK(cudaEventCreateWithFlags(e, cudaEventDisableTiming));
    return MD_OK;
}

}  // namespace

int md_stage_state(md_system *s, const double *xyz, const double *vxyz)
{
    if (!s || !xyz || !vxyz) { set_error("md_stage_state: null argument"); return MD_ERR_INVALID; }
    if (!is_pinned(xyz) || !is_pinned(vxyz)) { set_error("md_stage_state: the host arrays must be page-locked"); return MD_ERR_INVALID; }
    int rc = io_ready(s);
    if (rc) return rc;
    if (s->n_staged == 2) { set_error("md_stage_state: two states are staged already; md_commit_state takes the older one"); return MD_ERR_INVALID; }
    const size_t n3 = 3 * (size_t)s->P.N;
    const int slot = (s->in_head + s->n_staged) & 1;
    // a staging buffer is read on the system's stream only inside md_commit_state, which returns after that read
    double *dst = s->io_in[slot];
    if (vxyz == xyz + n3) {
        CK(cudaMemcpyAsync(dst, xyz, 2 * n3 * sizeof(double), cudaMemcpyHostToDevice, s->up_stream));
    } else {
        CK(cudaMemcpyAsync(dst, xyz, n3 * sizeof(double), cudaMemcpyHostToDevice, s->up_stream));
        CK(cudaMemcpyAsync(dst + n3, vxyz, n3 * sizeof(double), cudaMemcpyHostToDevice, s->up_stream));
    }
    CK(cudaEventRecord(s->ev_up[slot], s->up_stream));
    s->n_staged++;
    return MD_OK;
}

int md_commit_state(md_system *s)
{
    if (!s) { set_error("md_commit_state: null argument"); return MD_ERR_INVALID; }
    if (s->n_staged == 0) { set_error("md_commit_state: no staged state (md_stage_state first)"); return MD_ERR_INVALID; }
    const int slot = s->in_head;
    CK(cudaStreamWaitEvent(s->stream, s->ev_up[slot], 0));
    s->in_head ^= 1;
    s->n_staged--;
    return md_set_state_device(s, s->io_in[slot], s->io_in[slot] + 3 * (size_t)s->P.N);
}

int md_get_state_async(md_system *s, double *xyz, double *vxyz)
{
    if (!s || !xyz || !vxyz) { set_error("md_get_state_async: null argument"); return MD_ERR_INVALID; }
    if (!s->has_state) { set_error("no state loaded"); return MD_ERR_INVALID; }
    if (!is_pinned(xyz) || !is_pinned(vxyz)) { set_error("md_get_state_async: the host arrays must be page-locked"); return MD_ERR_INVALID; }
    int rc = io_ready(s);
    if (rc) return rc;
    const size_t n3 = 3 * (size_t)s->P.N;
    const int64_t d = s->n_down;
    double *src = s->io_out[d & 1];
    if (d >= 2) CK(cudaStreamWaitEvent(s->stream, s->ev_down[(d - 2) & 3], 0));      // the download before last read this buffer
    s->launches += 2;
    mdk_export(s->P, 0, src, s->stream);
    mdk_export(s->P, 1, src + n3, s->stream);
    CK(cudaEventRecord(s->ev_exported, s->stream));
    CK(cudaStreamWaitEvent(s->down_stream, s->ev_exported, 0));
    if (vxyz == xyz + n3) {
        CK(cudaMemcpyAsync(xyz, src, 2 * n3 * sizeof(double), cudaMemcpyDeviceToHost, s->down_stream));
    } else {
        CK(cudaMemcpyAsync(xyz, src, n3 * sizeof(double), cudaMemcpyDeviceToHost, s->down_stream));
        CK(cudaMemcpyAsync(vxyz, src + n3, n3 * sizeof(double), cudaMemcpyDeviceToHost, s->down_stream));
    }
    CK(cudaEventRecord(s->ev_down[d & 3], s->down_stream));
    s->n_down = d + 1;
    return MD_OK;
}

int md_wait_io(md_system *s, int32_t max_pending)
{
    if (!s) { set_error("md_wait_io: null argument"); return MD_ERR_INVALID; }
    if (max_pending < 0 || max_pending > 3) { set_error("md_wait_io: max_pending must be 0 .. 3"); return MD_ERR_INVALID; }
    if (!s->up_stream) return MD_OK;
    if (max_pending == 0) {
        CK(cudaStreamSynchronize(s->up_stream));
        CK(cudaStreamSynchronize(s->down_stream));
    } else if (s->n_down > max_pending) {
        // the copy stream runs the downloads in order: download n_down - max_pending - 1 complete => all before it too
        CK(cudaEventSynchronize(s->ev_down[(s->n_down - max_pending - 1) & 3]));
    }
    CK(cudaGetLastError());
    return MD_OK;
}

int md_measure_peaks(md_system *s, md_peaks *out)
{
    if (!s || !out) { set_error("md_measure_peaks: null argument"); return MD_ERR_INVALID; }
    memset(out, 0, sizeof(*out));
    int clk = 0;
    CK(cudaDeviceGetAttribute(&clk, cudaDevAttrClockRate, s->device));
    out->sm_count = s->sm_count;
    out->sm_clock_khz = clk;
    CK(cudaStreamSynchronize(s->stream));
    out->fp64_tflops = mdk_peak_fp64(s->stream, s->sm_count, s->P.partials);
    out->fp32_tflops = mdk_peak_fp32(s->stream, s->sm_count, s->P.partials);
    CK(cudaGetLastError());
    if (!(out->fp64_tflops > 0)) { set_error("md_measure_peaks: timing failed"); return MD_ERR_CUDA; }
    return MD_OK;
}

int md_set_bonds(md_system *s, int64_t n_bonds, const int32_t *ij, double k, double R0)
{
    if (!s || (n_bonds > 0 && !ij) || n_bonds < 0 || !(R0 > 0)) { set_error("md_set_bonds: bad argument"); return MD_ERR_INVALID; }
    if (!s->has_state) { set_error("md_set_bonds: load a state first"); return MD_ERR_INVALID; }
    if (s->stepped) { set_error("md_set_bonds: only before the first md_step"); return MD_ERR_INVALID; }
    MdDev &P = s->P;
    const size_t n = (size_t)P.N;
    std::vector<int> tab(2 * n, -1);
    int mx = 0;
    for (int64_t b = 0; b < n_bonds; b++) {
        const int i = ij[2 * b], j = ij[2 * b + 1];
        if (i < 0 || j < 0 || i >= P.N || j >= P.N || i == j) { set_error("md_set_bonds: bad pair (%d, %d)", i, j); return MD_ERR_INVALID; }
        if (i / P.N1 != j / P.N1) { set_error("md_set_bonds: pair (%d, %d) joins two independent systems", i, j); return MD_ERR_INVALID; }
        if (tab[i] == j || tab[n + i] == j) { set_error("md_set_bonds: pair (%d, %d) listed twice", i, j); return MD_ERR_INVALID; }
        for (int side = 0; side < 2; side++) {
            const int a = side ? j : i, c = side ? i : j;
            if (tab[a] < 0) tab[a] = c;
            else if (tab[n + a] < 0) tab[n + a] = c;
            else { set_error("md_set_bonds: atom %d has more than 2 bonds", a); return MD_ERR_UNSUPPORTED; }
            mx = std::max(mx, tab[n + a] >= 0 ? 2 : 1);
        }
    }
    if (s->P.rigid) { set_error("md_set_bonds: not with rigid molecules"); return MD_ERR_UNSUPPORTED; }
    if (!P.bond_orig) {
        P.bond_orig = (int *)dev_alloc(s, 2 * n * sizeof(int));
        P.bond_dev = (int *)dev_alloc(s, 2 * (size_t)P.N_pad * sizeof(int));
        if (!P.inv) P.inv = (int *)dev_alloc(s, n * sizeof(int));
        if (!P.bond_orig || !P.bond_dev || !P.inv) { set_error("device allocation failed"); return MD_ERR_NOMEM; }
    }
    CK(cudaMemcpyAsync(P.bond_orig, tab.data(), 2 * n * sizeof(int), cudaMemcpyHostToDevice, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    drop_graph(s);                 // the captured kernel arguments (MdDev by value) change
    P.has_bonds = n_bonds > 0;
    P.need_inv = 1;
    P.fene_k = k;
    P.fene_R02 = R0 * R0;
    P.fene_kf = (float)k;
    P.fene_R02f = (float)(R0 * R0);
    s->n_bonds_max = mx;
    // a rebuild fills inv / bond_dev for the current order, then forces are re-evaluated
    s->launches += 1;
    mdk_force_rebuild(P, s->stream);
    enqueue_rebuild(s);
    enqueue_forces_only(s);
    int rc = check_device_status(s);
    if (rc) return rc;
    CK(cudaMemsetAsync(&P.ctrl->n_rebuilds, 0, sizeof(int), s->stream));
    s->rebuilds_seen = 0;
    return MD_OK;
}

// Push-off of an overlapping chain start (include/md_b200.h; R12): initialisation, run in a temporary system.
int md_pushoff(md_system *s, const double *xyz, int64_t n_bonds, const int32_t *ij, double k, double R0,
               const md_pushoff_opts *opts, md_pushoff_report *report)
{
    if (!s || !xyz || n_bonds < 0 || (n_bonds > 0 && !ij) || !(R0 > 0)) { set_error("md_pushoff: bad argument"); return MD_ERR_INVALID; }
    md_pushoff_opts o;
    memset(&o, 0, sizeof(o));
    if (opts) o = *opts;
    if (!(o.r_cap_start > 0)) o.r_cap_start = 1.0;
    if (!(o.r_cap_end > 0)) o.r_cap_end = 0.8;
    if (o.ramp_steps <= 0) o.ramp_steps = 3000;
    if (o.max_steps <= 0) o.max_steps = 40000;
    if (o.check_interval <= 0) o.check_interval = 100;
    if (!(o.min_nonbonded > 0)) o.min_nonbonded = 0.85;
    if (!(o.max_bond > 0)) o.max_bond = 1.3;
    if (!(o.max_move > 0)) o.max_move = 0.05;
    if (!(o.temperature > 0)) o.temperature = 1.0;
    if (o.r_cap_end > o.r_cap_start || o.min_nonbonded >= s->prm.r_cut) { set_error("md_pushoff: bad options"); return MD_ERR_INVALID; }

    // temporary system: same box and model, global-index W built by the gathering kernel (no tile capacity to exceed),
    // twice the rows of W for the crowded start, split steps launched one by one
    md_params tp = s->prm;
    tp.lattice = MD_LATTICE_NONE;
    tp.precision = MD_PREC_F64;
    tp.force_variant = MD_FORCE_FULL_LIST;
    tp.step_mode = MD_STEP_SPLIT;
    tp.flags = MD_FLAG_GLOBAL_W | MD_FLAG_NO_GRAPH;
    tp.reorder_interval = 0;
    tp.stream = (void *)s->stream;
    tp.device = s->device;
    const size_t n3 = 3 * (size_t)s->P.N;
    std::vector<double> v(n3), r(n3);
    for (int b = 0; b < s->P.n_sys; b++)
        md_init_velocities(s->P.N1, o.temperature, o.seed + 1 + (uint64_t)b, v.data() + 3 * (size_t)b * s->P.N1);
    // Random walks cluster: the crowded start has atoms with several times the equilibrium number of neighbors
    // (73 against a mean of 18 at N = 2^20).  Start with 4 x the rows of W and double while the start overflows them.
    md_system *t = nullptr;
    int rc = MD_OK;
    for (int mult = 4; mult <= 32; mult *= 2) {
        tp.max_neighbors = mult * s->P.Mmax;
        const md_alloc_fn a0 = g_alloc; const md_free_fn f0 = g_free; void *u0 = g_alloc_user;
        g_alloc = s->alloc; g_free = s->free_; g_alloc_user = s->alloc_user;   // the temporary system allocates the way s does
        t = md_create_ex(&tp);
        g_alloc = a0; g_free = f0; g_alloc_user = u0;
        if (!t) return MD_ERR_CUDA;
        rc = upload_state(t, xyz, v.data(), true);
        if (rc != MD_ERR_NEBR_OVERFLOW) break;
        md_destroy(t);
        t = nullptr;
    }
    if (!t) return rc;
    unsigned long long *d_chk = nullptr, h_chk[2] = {0, 0};
    md_pushoff_report rep;
    memset(&rep, 0, sizeof(rep));
    auto bits_to_len = [](unsigned long long b) { double d; memcpy(&d, &b, sizeof(d)); return std::sqrt(d); };
    auto check = [&]() -> int {
        mdk_po_check(t->P, d_chk, t->stream);
        CK(cudaMemcpyAsync(h_chk, d_chk, sizeof(h_chk), cudaMemcpyDeviceToHost, t->stream));
        return check_device_status(t);
    };
    do {
        if (rc != MD_OK) break;
        if (n_bonds > 0 && (rc = md_set_bonds(t, n_bonds, ij, k, R0)) != MD_OK) break;
        d_chk = (unsigned long long *)dev_alloc(t, 2 * sizeof(unsigned long long));
        if (!d_chk) { set_error("md_pushoff: device allocation failed"); rc = MD_ERR_NOMEM; break; }
        if ((rc = check()) != MD_OK) break;
        rep.min_nonbonded_start = bits_to_len(h_chk[0]);
        const MdDev &P = t->P;
        const double ke_target = 1.5 * (double)(P.N - P.n_sys) * o.temperature;
        const double vlim = o.max_move / P.dt;
        double rcap = o.r_cap_start;
        mdk_po_force(P, rcap * rcap, t->stream);
        bool done = false;
        int64_t step = 0;
        while (!done && step < o.max_steps) {
            for (int c = 0; c < o.check_interval; c++, step++) {
                const double x = std::min(1.0, (double)step / o.ramp_steps);
                rcap = o.r_cap_start + x * (o.r_cap_end - o.r_cap_start);
                mdk_po_kick_drift(P, rcap * rcap, vlim * vlim, ke_target, step == 0, t->stream);
                mdk_decide(P, false, t->stream, 0ull);
                enqueue_rebuild(t);
                mdk_po_force(P, rcap * rcap, t->stream);
                mdk_po_kick(P, t->stream);
            }
            t->launches += 12 * (int64_t)o.check_interval;
            if ((rc = check()) != MD_OK) break;
            rep.min_nonbonded = bits_to_len(h_chk[0]);
            rep.max_bond = bits_to_len(h_chk[1]);
            done = step >= o.ramp_steps && rep.min_nonbonded > o.min_nonbonded && (n_bonds == 0 || rep.max_bond < o.max_bond);
        }
        rep.steps = step;
        if (rc != MD_OK) break;
        if (!done) {
            set_error("md_pushoff: after %lld steps the smallest non-bonded distance is %.4f (want > %.3f) and the longest bond %.4f (want < %.3f)",
                      (long long)step, rep.min_nonbonded, o.min_nonbonded, rep.max_bond, o.max_bond);
            rc = MD_ERR_UNSUPPORTED;
            break;
        }
        if ((rc = download(t, 0, r.data())) != MD_OK) break;
    } while (0);
    s->launches += t->launches;
    md_destroy(t);
    if (report) *report = rep;
    if (rc != MD_OK) return rc;
    for (int b = 0; b < s->P.n_sys; b++)
        md_init_velocities(s->P.N1, o.temperature, o.seed + (uint64_t)b, v.data() + 3 * (size_t)b * s->P.N1);
    if ((rc = upload_state(s, r.data(), v.data(), true)) != MD_OK) return rc;
    return n_bonds > 0 ? md_set_bonds(s, n_bonds, ij, k, R0) : MD_OK;
}

// ---- rigid molecules (R20) ----
int md_set_rigid(md_system *s, int32_t n_sites, const double *body_xyz)
{
    if (!s || !body_xyz || n_sites < 3 || n_sites > 8) { set_error("md_set_rigid: 3 .. 8 sites per molecule"); return MD_ERR_INVALID; }
    MdDev &P = s->P;
    if (P.sp || P.half_list || P.tiled || P.n_sys > 1 || P.has_bonds || P.layer_H || P.w_col != 1) {
        set_error("md_set_rigid: fp64, full-list forces, global-index W (MD_FLAG_GATHER_W for long columns), one system, no bonds");
        return MD_ERR_UNSUPPORTED;
    }
    if (P.N % n_sites) { set_error("md_set_rigid: n_atoms is not a multiple of the sites per molecule"); return MD_ERR_INVALID; }
    // unit-mass sites: centre of mass at the origin, inertia tensor diagonal with positive moments (principal frame)
    double I[3][3] = {{0}}, com[3] = {0, 0, 0}, bmax = 0.0;
    for (int k = 0; k < n_sites; k++) {
        const double *b = body_xyz + 3 * k, b2 = b[0] * b[0] + b[1] * b[1] + b[2] * b[2];
        bmax = std::max(bmax, sqrt(b2));
        for (int r = 0; r < 3; r++) {
            com[r] += b[r];
            for (int c = 0; c < 3; c++) I[r][c] += (r == c ? b2 : 0.0) - b[r] * b[c];
        }
    }
    const double tol = 1e-12 * (I[0][0] + I[1][1] + I[2][2] + 1.0);
    bool bad = fabs(com[0]) + fabs(com[1]) + fabs(com[2]) > 1e-12 * n_sites * (bmax + 1.0);
    for (int r = 0; r < 3; r++)
        for (int c = 0; c < 3; c++)
            if ((r != c && fabs(I[r][c]) > tol) || (r == c && !(I[r][c] > 0))) bad = true;
    if (bad) { set_error("md_set_rigid: give the sites in the principal frame about their centre of mass (all three moments > 0)"); return MD_ERR_INVALID; }
    drop_graph(s);
    P.rb_ns = n_sites;
    P.rb_nm = P.N / n_sites;
    for (int k = 0; k < 3 * n_sites; k++) P.rb_body[k] = body_xyz[k];
    P.rb_M = (double)n_sites;
    P.rb_bmax = bmax;
    P.rb_Imin = std::min(I[0][0], std::min(I[1][1], I[2][2]));
    for (int c = 0; c < 3; c++) P.rb_I[c] = I[c][c];
    if (!P.rb_R) {
        const size_t nm = (size_t)P.rb_nm;
        P.rb_R = (double *)dev_alloc(s, 3 * nm * sizeof(double)); P.rb_V = (double *)dev_alloc(s, 3 * nm * sizeof(double));
        P.rb_A = (double *)dev_alloc(s, 9 * nm * sizeof(double)); P.rb_pi = (double *)dev_alloc(s, 3 * nm * sizeof(double));
        P.rb_off = (double *)dev_alloc(s, 3 * (size_t)P.N * sizeof(double));
        if (!P.inv) P.inv = (int *)dev_alloc(s, (size_t)P.N * sizeof(int));
        if (!P.rb_R || !P.rb_V || !P.rb_A || !P.rb_pi || !P.rb_off || !P.inv) { set_error("device allocation failed"); return MD_ERR_NOMEM; }
    }
    P.rigid = 1;
    s->persist = false;
    P.need_inv = 1;
    P.tile_build = 0;          // the gathering build kernel knows the molecules (sites of one molecule are no neighbors)
    s->has_state = false;      // load the molecules with md_set_rigid_state
    return MD_OK;
}

int md_set_rigid_state(md_system *s, const double *com, const double *rot, const double *vcom, const double *angmom_body)
{
    if (!s || !com || !rot || !vcom || !angmom_body) { set_error("md_set_rigid_state: null argument"); return MD_ERR_INVALID; }
    MdDev &P = s->P;
    if (!P.rigid) { set_error("md_set_rigid_state: call md_set_rigid first"); return MD_ERR_INVALID; }
    const size_t nm = (size_t)P.rb_nm;
    const int ns = P.rb_ns;
    const double L = P.L;
    std::vector<double> xyz(3 * (size_t)P.N), v(3 * (size_t)P.N);
    for (size_t m = 0; m < nm; m++) {
        const double *A = rot + 9 * m, *R = com + 3 * m, *V = vcom + 3 * m, *pi = angmom_body + 3 * m;
        const double w[3] = {pi[0] / P.rb_I[0], pi[1] / P.rb_I[1], pi[2] / P.rb_I[2]};
        for (int k = 0; k < ns; k++) {
            const double *b = P.rb_body + 3 * k;
            const double u[3] = {w[1] * b[2] - w[2] * b[1], w[2] * b[0] - w[0] * b[2], w[0] * b[1] - w[1] * b[0]};
            for (int c = 0; c < 3; c++) {
                double x = R[c] + (A[3 * c] * b[0] + A[3 * c + 1] * b[1] + A[3 * c + 2] * b[2]);
                if (!std::isfinite(x)) { set_error("md_set_rigid_state: non-finite state"); return MD_ERR_NONFINITE; }
                x -= L * floor(x / L);
                if (x >= L || x < 0.0) x = 0.0;
                xyz[3 * (m * ns + k) + c] = x;
                v[3 * (m * ns + k) + c] = V[c] + (A[3 * c] * u[0] + A[3 * c + 1] * u[1] + A[3 * c + 2] * u[2]);
            }
        }
    }
    CK(cudaMemcpyAsync(P.rb_R, com, 3 * nm * sizeof(double), cudaMemcpyHostToDevice, s->stream));
    CK(cudaMemcpyAsync(P.rb_A, rot, 9 * nm * sizeof(double), cudaMemcpyHostToDevice, s->stream));
    CK(cudaMemcpyAsync(P.rb_V, vcom, 3 * nm * sizeof(double), cudaMemcpyHostToDevice, s->stream));
    CK(cudaMemcpyAsync(P.rb_pi, angmom_body, 3 * nm * sizeof(double), cudaMemcpyHostToDevice, s->stream));
    CK(cudaMemsetAsync(P.rb_off, 0, 3 * (size_t)P.N * sizeof(double), s->stream));
    CK(cudaStreamSynchronize(s->stream));       // the host arrays may be pageable and go out of scope
    return upload_state(s, xyz.data(), v.data(), true);
}

int md_get_rigid_state(md_system *s, double *com, double *rot, double *vcom, double *angmom_body)
{
    if (!s || !com || !rot || !vcom || !angmom_body) { set_error("md_get_rigid_state: null argument"); return MD_ERR_INVALID; }
    const MdDev &P = s->P;
    if (!P.rigid || !s->has_state) { set_error("md_get_rigid_state: no rigid state"); return MD_ERR_INVALID; }
    const size_t nm = (size_t)P.rb_nm;
    CK(cudaMemcpyAsync(com, P.rb_R, 3 * nm * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaMemcpyAsync(rot, P.rb_A, 9 * nm * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaMemcpyAsync(vcom, P.rb_V, 3 * nm * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaMemcpyAsync(angmom_body, P.rb_pi, 3 * nm * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    return MD_OK;
}

int md_set_angles(md_system *s, double k_theta, double cos_theta0)
{
    if (!s || !(k_theta >= 0) || !(cos_theta0 >= -1.0 && cos_theta0 <= 1.0)) { set_error("md_set_angles: bad argument"); return MD_ERR_INVALID; }
    if (!s->P.has_bonds) { set_error("md_set_angles: set the bond list first"); return MD_ERR_INVALID; }
    if (s->stepped) { set_error("md_set_angles: only before the first md_step"); return MD_ERR_INVALID; }
    if (s->P.tiled) { set_error("md_set_angles: global-index W layouts only (use MD_FLAG_GATHER_W)"); return MD_ERR_UNSUPPORTED; }
    drop_graph(s);                 // the captured kernel arguments (MdDev by value) change
    s->P.has_angles = k_theta > 0;
    s->persist = s->persist && mdk_persist_ok(s->P);
    s->P.ang_k = k_theta;
    s->P.ang_c0 = cos_theta0;
    enqueue_forces_only(s);
    return check_device_status(s);
}

int md_set_dihedrals(md_system *s, double k_phi, double cos_phi0)
{
    if (!s || !(k_phi >= 0) || !(cos_phi0 >= -1.0 && cos_phi0 <= 1.0)) { set_error("md_set_dihedrals: bad argument"); return MD_ERR_INVALID; }
    if (!s->P.has_bonds) { set_error("md_set_dihedrals: set the bond list first"); return MD_ERR_INVALID; }
    if (s->stepped) { set_error("md_set_dihedrals: only before the first md_step"); return MD_ERR_INVALID; }
    if (s->P.tiled) { set_error("md_set_dihedrals: global-index W layouts only (use MD_FLAG_GATHER_W)"); return MD_ERR_UNSUPPORTED; }
    drop_graph(s);
    s->P.has_dihedrals = k_phi > 0;
    s->persist = s->persist && mdk_persist_ok(s->P);
    s->P.dih_k = k_phi;
    s->P.dih_c0 = cos_phi0;
    enqueue_forces_only(s);
    return check_device_status(s);
}

int md_rebuild_neighbors(md_system *s)
{
    if (!s || !s->has_state) { set_error("md_rebuild_neighbors: no state"); return MD_ERR_INVALID; }
    s->launches += 1;
    mdk_force_rebuild(s->P, s->stream);
    enqueue_rebuild(s);
    enqueue_forces_only(s);
    return check_device_status(s);
}

int md_step(md_system *s, int64_t n)
{
    if (!s || n < 0) { set_error("md_step: bad argument"); return MD_ERR_INVALID; }
    if (!s->has_state) { set_error("md_step: no state loaded (lattice NONE needs md_set_state)"); return MD_ERR_INVALID; }
    if (n == 0) return MD_OK;
    s->stepped = true;
    const MdDev &P = s->P;
    cudaStream_t st = s->stream;
    if (P.rigid) {
        // rigid molecules: per-molecule half kick + free rotation + drift, rebuild decision, site forces, half kick
        for (int64_t k = 0; k < n; k++) {
            { Timed t(s, MD_T_INTEGRATE, 1); mdk_rigid_kick_drift(P, st); }
            { Timed t(s, MD_T_DECIDE, 1); mdk_decide(P, false, st, 0ull); }
            enqueue_rebuild(s);
            enqueue_forces_only(s);
            { Timed t(s, MD_T_INTEGRATE, 1); mdk_rigid_kick(P, st); }
        }
        s->step += n;
        return check_device_status(s);
    }
    if (s->persist && !s->profiling) {
        // small system: one cooperative launch whose blocks stay resident over all n steps (md_kernels.cu: k_persist)
        if (mdk_persist_steps(P, (long long)n, st) != 0) {
            cudaGetLastError();
            s->persist = false;                         // e.g. the device is shared and the grid no longer fits: step graph
        } else {
            s->launches += 1;
            s->step += n;
            return check_device_status(s);
        }
    }
    if (s->prm.step_mode == MD_STEP_FUSED) {
        // leapfrog form: opening half kick + drift, (n-1) fused force+kick+drift kernels, closing force + half kick
        const bool graphs = have_graphs(s);
        if (graphs) {
            CK(cudaGraphLaunch(s->gexec[0], st));
            int64_t k = 1;
            for (; k + GRAPH_UNROLL <= n; k += GRAPH_UNROLL) CK(cudaGraphLaunch(s->gexec[2], st));
            for (; k < n; k++) CK(cudaGraphLaunch(s->gexec[1], st));
            s->graph_steps += n;
            s->launches += 2 + (n - 1) * 2;               // + the rebuild chains, added in check_device_status
        } else {
            { Timed t(s, MD_T_INTEGRATE, 1); mdk_kick_drift(P, s->lc, st); }
            enqueue_decide(s, false);
            enqueue_rebuild(s);
            for (int64_t k = 1; k < n; k++) {
                { Timed t(s, MD_T_FUSED_STEP, 1); enqueue_force(s, 1); }
                enqueue_decide(s, true);
                enqueue_rebuild(s);
            }
        }
        { Timed t(s, MD_T_FORCE, 1); enqueue_force(s, 2); }
    } else {
        const bool graphs = have_graphs(s);
        for (int64_t k = 0; k < n; k++) {
            if (graphs) {
                CK(cudaGraphLaunch(s->gexec[0], st));
                s->graph_steps += 1;
                s->launches += 2;
            } else {
                { Timed t(s, MD_T_INTEGRATE, 1); mdk_kick_drift(P, s->lc, st); }
                enqueue_decide(s, false);
                enqueue_rebuild(s);
            }
            enqueue_forces_only(s);
            { Timed t(s, MD_T_INTEGRATE, 1); mdk_kick(P, s->lc, st); }
        }
    }
    s->step += n;
    return check_device_status(s);
}

int md_energies(md_system *s, md_energy *out)
{
    if (!s || !out) { set_error("md_energies: null argument"); return MD_ERR_INVALID; }
    if (!s->has_state) { set_error("md_energies: no state"); return MD_ERR_INVALID; }
    { Timed t(s, MD_T_ENERGY, 1); if (s->P.tiled) mdk_tile_energy(s->P, s->stream); else mdk_energy(s->P, s->lc, s->stream); }
    int rc = check_device_status(s);
    if (rc) return rc;
    const DevCtrl &c = *s->h_ctrl;
    out->ke = c.red[RED_KE];
    out->pe_pair = c.red[RED_PE];
    out->pe_bond = c.red[RED_PEB];
    out->virial = c.red[RED_VIR];
    out->px = c.red[RED_PX]; out->py = c.red[RED_PY]; out->pz = c.red[RED_PZ];
    out->vmax = sqrt(c.red[RED_VMAX2]);
    out->step = s->step;
    out->n_rebuilds = c.n_rebuilds;
    out->max_neighbors = c.max_nnb;
    out->max_cell_occupancy = c.max_occ;
    out->mean_neighbors = (double)c.nnb_total * (s->P.half_list ? 2.0 : 1.0) / (double)s->P.N;
    if (!std::isfinite(out->ke + out->pe_pair + out->pe_bond)) { set_error("non-finite energy"); return MD_ERR_NONFINITE; }
    return MD_OK;
}

int md_get_positions(md_system *s, double *xyz) { return download(s, 0, xyz); }
int md_get_velocities(md_system *s, double *xyz) { return download(s, 1, xyz); }
int md_get_forces(md_system *s, double *xyz) { return download(s, 2, xyz); }

int md_get_positions_device(md_system *s, double *xyz_device) { return export_device(s, 0, xyz_device); }
int md_get_velocities_device(md_system *s, double *xyz_device) { return export_device(s, 1, xyz_device); }
int md_get_forces_device(md_system *s, double *xyz_device) { return export_device(s, 2, xyz_device); }

// positions and velocities in one call: two export kernels, one device-to-host transfer when the two host arrays are
// adjacent (vxyz == xyz + 3N), one synchronisation
int md_get_state(md_system *s, double *xyz, double *vxyz)
{
    if (!s || !xyz || !vxyz) { set_error("md_get_state: null argument"); return MD_ERR_INVALID; }
    if (!s->has_state) { set_error("no state loaded"); return MD_ERR_INVALID; }
    const size_t n3 = 3 * (size_t)s->P.N;
    s->launches += 2;
    mdk_export(s->P, 0, s->P.scratch, s->stream);
    mdk_export(s->P, 1, s->P.scratch + n3, s->stream);
    const bool direct = is_pinned(xyz) && is_pinned(vxyz);
    if (direct && vxyz == xyz + n3) {
        CK(cudaMemcpyAsync(xyz, s->P.scratch, 2 * n3 * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    } else {
        CK(cudaMemcpyAsync(direct ? xyz : s->h_stage, s->P.scratch, n3 * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
        CK(cudaMemcpyAsync(direct ? vxyz : s->h_stage + n3, s->P.scratch + n3, n3 * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    }
    CK(cudaStreamSynchronize(s->stream));
    CK(cudaGetLastError());
    if (!direct) { memcpy(xyz, s->h_stage, n3 * sizeof(double)); memcpy(vxyz, s->h_stage + n3, n3 * sizeof(double)); }
    return MD_OK;
}

int md_get_neighbors(md_system *s, int32_t *counts, int32_t *list, int32_t *max_neighbors_out)
{
    if (!s || !counts) { set_error("md_get_neighbors: null argument"); return MD_ERR_INVALID; }
    if (!s->has_state) { set_error("md_get_neighbors: no state"); return MD_ERR_INVALID; }
    int rc = fetch_ctrl(s);
    if (rc) return rc;
    const MdDev &P = s->P;
    const int N = P.N, M = P.Mmax;
    const size_t np = (size_t)P.N_pad;
    const int nrows = std::min(M, std::max(1, s->h_ctrl->max_nnb));
    const int rows = P.tiled ? (nrows + 1) / 2 : (P.w_col == 1 ? nrows : M);      // tiled: two 16-bit entries per 32-bit word
    std::vector<int> nnb(N), id(N), W((size_t)rows * np);
    CK(cudaMemcpy(nnb.data(), P.nnb, N * sizeof(int), cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(id.data(), P.id[s->h_ctrl->v_dst], N * sizeof(int), cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(W.data(), P.W, (size_t)rows * np * sizeof(int), cudaMemcpyDeviceToHost));
    if (max_neighbors_out) *max_neighbors_out = M;
    std::vector<int> cnt(N, 0);
    bool overflow = false;
    auto add = [&](int a, int b) {
        if (cnt[a] < M) { if (list) list[(size_t)a * M + cnt[a]] = b; }
        else overflow = true;
        cnt[a]++;
    };
    if (P.tiled) {
        // rebuild every block's tile layout from cell_start exactly as the kernels do (md_tile.cu: tile_setup)
        std::vector<int> cs((size_t)P.NC + 1), map;
        CK(cudaMemcpy(cs.data(), P.cell_start, cs.size() * sizeof(int), cudaMemcpyDeviceToHost));
        const int nblocks = P.tg.nsx * P.tg.nsy * P.tg.nsz * P.tg.nsys;
        for (int b = 0; b < nblocks; b++) {
            const TileBox B = tile_box(P.tg, P.nc, P.ncx, b);
            map.clear();
            std::vector<std::pair<int, int>> own;            // (global start, length) of the box's own rows
            for (int q = 0; q < B.nq; q++) {
                int rowc, ysh, zsh, xa, xc;
                tile_row(B, P.nc, P.ncx, P.kx, q, rowc, ysh, zsh, xa, xc);
                const int g[3] = {cs[rowc + xa], cs[rowc + B.x0], cs[rowc + xc]};
                const int n[3] = {cs[rowc + xa + P.kx] - g[0], cs[rowc + B.x0 + B.sxc] - g[1], cs[rowc + xc + P.kx] - g[2]};
                for (int k = 0; k < 3; k++) for (int u = 0; u < n[k]; u++) map.push_back(g[k] + u);
                const int qy = q % B.nyq, qz = q / B.nyq;
                if (qy >= 1 && qy <= B.ny && qz >= 1 && qz <= B.nz) own.push_back({g[1], n[1]});
            }
            for (auto &r : own)
                for (int pidx = r.first; pidx < r.first + r.second; pidx++)
                    for (int m = 0; m < nnb[pidx]; m++) {
                        const unsigned w2 = (unsigned)W[(size_t)(m >> 1) * np + pidx];
                        const unsigned e = (m & 1) ? (w2 >> 16) : (w2 & 0xffffu);
                        const unsigned l = e & T_INDEX_MASK;
                        if (l >= map.size()) { set_error("md_get_neighbors: corrupt tile index"); return MD_ERR_INVALID; }
                        add(id[pidx], id[map[l]]);
                    }
        }
    } else {
        for (int p = 0; p < N; p++)
            for (int m = 0; m < nnb[p]; m++) {
                const int i = id[p], j = id[(unsigned)W[(size_t)m * P.w_row + (size_t)p * P.w_col] & 0x1fffffffu];   // top 3 bits: image flags
                add(i, j);
                if (P.half_list) add(j, i);
            }
    }
    for (int i = 0; i < N; i++) {
        counts[i] = cnt[i];
        if (list) for (int m = std::min(cnt[i], M); m < M; m++) list[(size_t)i * M + m] = -1;
    }
    if (overflow) { set_error("md_get_neighbors: symmetrised list exceeds Mmax"); return MD_ERR_NEBR_OVERFLOW; }
    return MD_OK;
}

int md_get_info(md_system *s, md_info *out)
{
    if (!s || !out) { set_error("md_get_info: null argument"); return MD_ERR_INVALID; }
    memset(out, 0, sizeof(*out));
    out->n_atoms = s->P.N1; out->n_pad = s->P.N_pad; out->n_systems = s->P.n_sys;
    out->box = s->P.L; out->r_neighbor = s->r_n; out->cell_width = s->cell_w;
    out->cells_per_edge = s->P.nc; out->max_neighbors = s->P.Mmax; out->block_size = s->lc.block;
    out->force_variant = s->prm.force_variant; out->step_mode = s->prm.step_mode;
    out->n_bonds_per_atom_max = s->n_bonds_max;
    out->w_layout = s->P.tiled ? MD_W_TILED : MD_W_GLOBAL;
    if (s->P.tile_build) {
        out->tile_cells[0] = s->P.tg.S / s->P.kx; out->tile_cells[1] = s->P.tg.R; out->tile_cells[2] = s->P.tg.RZ;
        out->tile_capacity = s->P.tg.cap; out->tile_threads = s->P.tg.threads;
    }
    out->use_graph = s->persist ? 2 : (s->gexec[0] ? 1 : 0);
    out->precision = s->prm.precision;
    out->n_layers = s->P.n_layers;
    out->cells_x = s->P.ncx; out->cell_split_x = s->P.kx; out->sm_count = s->sm_count;
    // counted by the last neighbor build (as of the last status read); before any: 9 rows of 2 kx + 1 fine cells, an
    // upper bound (rows far from the atom are scanned over a shorter window or not at all)
    out->candidates_per_atom = s->h_ctrl && s->h_ctrl->cand_total ? (double)s->h_ctrl->cand_total / (double)s->P.N
                                                                  : 9.0 * (2.0 * s->P.kx + 1.0) * (double)s->P.N1 / (double)s->P.NC1;
    out->device_bytes = s->bytes;
    out->kernel_launches = s->launches;
    snprintf(out->device_name, sizeof(out->device_name), "%s", s->device_name);
    return MD_OK;
}

int md_set_profiling(md_system *s, int enabled)
{
    if (!s) { set_error("null system"); return MD_ERR_INVALID; }
    s->profiling = enabled != 0;
    return MD_OK;
}

int md_get_timers(md_system *s, double *ms, int64_t *launches)
{
    if (!s) { set_error("null system"); return MD_ERR_INVALID; }
    CK(cudaStreamSynchronize(s->stream));
    resolve_timers(s);
    for (int k = 0; k < MD_T_COUNT; k++) {
        if (ms) ms[k] = s->t_ms[k];
        if (launches) launches[k] = s->t_n[k];
    }
    return MD_OK;
}

int md_reset_timers(md_system *s)
{
    if (!s) { set_error("null system"); return MD_ERR_INVALID; }
    CK(cudaStreamSynchronize(s->stream));
    resolve_timers(s);
    for (int k = 0; k < MD_T_COUNT; k++) { s->t_ms[k] = 0; s->t_n[k] = 0; }
    return MD_OK;
}

}  // extern "C"

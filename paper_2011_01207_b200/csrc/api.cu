// api.cu -- the C ABI of libtkhp (include/tkhp.h): parameter checks, workspace carve,
// context life cycle, phase timing and the host-buffer end-to-end entry.
#include <math.h>
#include <new>

#include "common.cuh"

namespace tkhp {

static thread_local char g_create_err[512] = "";

// for the entry points that have no context (energy_static.cu): the text tkhp_last_error(NULL) returns
void set_thread_error(const char *msg) { snprintf(g_create_err, sizeof(g_create_err), "%s", msg); }

static int grid_bits_for(double extent) {
    int b = 1;
    while (extent / (double)(1 << b) > 2.5 && b < 8) ++b;
    return b;
}

static int check_params(const tkhp_params *p, char *err, size_t n) {
    if (!p) { snprintf(err, n, "params is NULL"); return TKHP_EINVAL; }
    if (p->n_atoms < 1) { snprintf(err, n, "n_atoms must be >= 1"); return TKHP_EINVAL; }
    if (p->precision != TKHP_FP64 && p->precision != TKHP_MIXED && p->precision != TKHP_FIXED) { snprintf(err, n, "bad precision"); return TKHP_EINVAL; }
    if (p->list_mode != TKHP_LIST_TILES && p->list_mode != TKHP_LIST_CLUSTER && p->list_mode != TKHP_LIST_ATOM) { snprintf(err, n, "bad list_mode"); return TKHP_EINVAL; }
    if (!(p->cutoff > 0.0) || !(p->skin >= 0.0) || !isfinite(p->cutoff) || !isfinite(p->skin)) { snprintf(err, n, "cutoff must be > 0 and skin >= 0"); return TKHP_EINVAL; }
    if (!(p->ewald_beta >= 0.0) || !isfinite(p->ewald_beta)) { snprintf(err, n, "ewald_beta must be >= 0"); return TKHP_EINVAL; }
    if (!(p->thole_a > 0.0) || !isfinite(p->thole_a)) { snprintf(err, n, "thole_a must be > 0"); return TKHP_EINVAL; }
    if (!isfinite(p->box)) { snprintf(err, n, "box must be finite"); return TKHP_EINVAL; }
    if (p->box > 0.0 && p->cutoff + p->skin > 0.5 * p->box) {
        snprintf(err, n, "cutoff + skin = %g exceeds box/2 = %g (single minimum image)", p->cutoff + p->skin, 0.5 * p->box);
        return TKHP_ECUTOFF;
    }
    if (p->ewald_beta * p->cutoff > 6.0) {
        snprintf(err, n, "ewald_beta * cutoff must be <= 6 (range of the erfc fits)");
        return TKHP_EINVAL;
    }
    if (p->precision != TKHP_FP64 && p->n_atoms > (1 << 24)) { snprintf(err, n, "MIXED / FIXED precision supports up to 2^24 atoms"); return TKHP_EINVAL; }
    if (p->max_tiles_per_block < 0 || p->max_nbrs_per_cluster < 0 || p->max_nbrs_per_atom < 0) { snprintf(err, n, "negative capacity"); return TKHP_EINVAL; }
    if (p->solver_flags & ~(TKHP_SOLVER_NO_PERSISTENT | TKHP_SOLVER_NO_FUSED_STEP | TKHP_SOLVER_STORED_T | TKHP_SOLVER_TEST_BARRIER_FAULT) || p->reserved != 0) { snprintf(err, n, "unknown solver_flags / non-zero reserved field"); return TKHP_EINVAL; }
    if (p->max_stage_per_chunk < 0 || (p->max_stage_per_chunk & 31)) { snprintf(err, n, "max_stage_per_chunk must be a non-negative multiple of 32"); return TKHP_EINVAL; }
    return TKHP_OK;
}

static long long tile_capacity(const tkhp_params *p, int n_blocks) {
    const long long all = (long long)n_blocks * (n_blocks + 1) / 2;
    long long per_block;
    if (p->max_tiles_per_block > 0) {
        per_block = p->max_tiles_per_block;
    } else if (p->box > 0.0) {
        // uniform-density estimate: blocks whose boxes come within reach of a block's box fill a cube
        // of edge 2 reach + 2 e (e = edge of a 32-atom cube, widened 1.35x for box overlap); half list.
        const double vol = p->box * p->box * p->box;
        const double rho = p->n_atoms / vol;
        const double e = 1.35 * cbrt(32.0 / rho);
        double edge = 2.0 * (p->cutoff + p->skin) + 2.0 * e;
        if (edge > p->box) edge = p->box;
        per_block = (long long)(1.6 * 0.5 * edge * edge * edge * rho / 32.0) + 16;
    } else {
        per_block = 4096;
    }
    long long cap = per_block * n_blocks;
    if (cap > all) cap = all;
    if (cap < 1) cap = 1;
    return cap;
}

// One function lays out the workspace for both the size query and the real carve.
static size_t carve(Ctx *c, const tkhp_params *p, void *base) {
    Carver w(base);
    const size_t n = p->n_atoms;
    const int n_blocks = (int)((n + BLOCK - 1) / BLOCK);
    const size_t n_pad = (size_t)n_blocks * BLOCK;
    const int n_super = (n_blocks + SUPER - 1) / SUPER;
    const int b_alloc = p->box > 0.0 ? grid_bits_for(p->box) : 6;      // open boundary: b <= 6
    size_t n_cells = (size_t)1 << (3 * b_alloc);
    size_t bins = n_cells > n ? n_cells : n;
    const long long cap_tiles = tile_capacity(p, n_blocks);
    const bool f64 = p->precision == TKHP_FP64;

    Ctx dummy;
    Ctx *o = c ? c : &dummy;
    o->n = (int)n; o->n_blocks = n_blocks; o->n_pad = (int)n_pad; o->n_super = n_super;
    o->n_cells_alloc = (int)n_cells; o->cap_tiles = cap_tiles;
    o->grid_bits_host = p->box > 0.0 ? b_alloc : -1;

    o->st = w.take<DeviceState>(1);
    o->key = w.take<uint32_t>(n);
    o->cell_count = w.take<uint32_t>(bins + 2);
    o->cell_start = w.take<uint32_t>(n_cells + 2);
    o->scan_tmp = w.take<uint32_t>((bins + 2) / 2048 + 2);
    o->tmp_idx = w.take<int32_t>(n);
    o->key2 = w.take<uint32_t>(n);
    o->count2 = w.take<uint32_t>(n + 2);
    o->scan_tmp2 = w.take<uint32_t>((n + 2) / 2048 + 2);
    o->tmp_idx2 = w.take<int32_t>(n);
    o->perm = w.take<int32_t>(n_pad);
    o->pos_o = w.take<double>(3 * n);
    o->group_o = w.take<int32_t>(n);
    o->grp_start = w.take<uint32_t>(n + 2);
    o->grp_members = w.take<int32_t>(n);
    o->xyzw32 = w.take<float4>(n_pad);
    o->xyzw64 = f64 ? w.take<double4>(n_pad) : nullptr;
    o->bcentre = w.take<double4>(n_blocks);
    o->bhalf = w.take<double4>(n_blocks);
    o->scentre = w.take<double4>(n_super);
    o->shalf = w.take<double4>(n_super);
    o->alpha_s = w.take<double>(n_pad);
    o->inv_alpha_s = w.take<double>(n_pad);
    o->row_count = w.take<uint32_t>(n_blocks + 2);
    o->row_start = w.take<uint32_t>(n_blocks + 2);
    o->pairs = w.take<int2>((size_t)cap_tiles);
    o->acc = w.take<double>(3 * n_pad);
    o->mu32 = f64 ? nullptr : w.take<float4>(n_pad);
    o->u32 = f64 ? nullptr : w.take<float4>(n_pad);
    o->mu64 = f64 ? w.take<double4>(n_pad) : nullptr;
    o->mp32 = f64 ? nullptr : w.take<float4>(3 * n_pad);
    o->mp64 = f64 ? w.take<double4>(3 * n_pad) : nullptr;
    o->vE = w.take<double>(3 * n_pad);
    o->vmu = w.take<double>(3 * n_pad);
    o->vr = w.take<double>(3 * n_pad);
    o->vp = w.take<double>(3 * n_pad);
    o->vq = w.take<double>(3 * n_pad);
    o->part_cap = n_blocks + MAX_PARTIALS;
    o->partials = w.take<double>(6 * (size_t)o->part_cap);
    // staging for the host-buffer entry
    o->h_pos = w.take<double>(3 * n);
    o->h_alpha = w.take<double>(n);
    o->h_group = w.take<int32_t>(n);
    o->h_charge = w.take<double>(n);
    o->h_dipole = w.take<double>(3 * n);
    o->h_quad = w.take<double>(6 * n);
    o->h_field = w.take<double>(3 * n);
    o->h_mu = w.take<double>(3 * n);
    o->h_energy = w.take<double>(1);
    {
        const size_t tb = atom_stored_bytes(p, n_blocks);
        o->tstore = tb ? w.take<uint4>(tb / sizeof(uint4)) : nullptr;
        o->stored_t = tb != 0;
    }
    o->cl_ws_bytes = cluster_workspace_bytes(p, n_blocks);
    o->cl_ws = w.take<char>(o->cl_ws_bytes);
    w.take<char>(256);
    return w.off;
}

int ensure_header(Ctx *c, cudaStream_t s) {
    if (!c->built) return set_err(c, TKHP_ENOLIST, "tkhp_nblist_build() has not been called%s");
    if (!c->header_valid) {
        TKHP_CUDA(c, cudaMemcpyAsync(c->h_state, c->st, sizeof(DeviceState), cudaMemcpyDeviceToHost, s));
        TKHP_CUDA(c, cudaStreamSynchronize(s));
        c->header_valid = true;
        c->n_tiles_host = c->h_state->n_tiles;
        c->list_mode_in_use = TKHP_LIST_TILES;
        if (c->p.list_mode != TKHP_LIST_TILES && !c->h_state->cluster_bad)
            c->list_mode_in_use = (c->p.list_mode == TKHP_LIST_ATOM && !c->h_state->atom_bad) ? TKHP_LIST_ATOM : TKHP_LIST_CLUSTER;
    }
    const DeviceState &h = *c->h_state;
    if (h.err_nonfinite) return set_err(c, TKHP_ENONFINITE, "non-finite position passed to tkhp_nblist_build%s");
    if (h.err_bad_alpha) return set_err(c, TKHP_ENONFINITE, "polarizability <= 0 or non-finite%s");
    if (h.err_bad_group) return set_err(c, TKHP_EINVAL, "group id outside [0, n_atoms)%s");
    if (h.err_capacity) return set_err(c, TKHP_ECAPACITY, "neighbour list exceeds the workspace capacity (raise max_tiles_per_block / max_nbrs_per_cluster)%s");
    return TKHP_OK;
}

static void tic(Ctx *c, int phase, cudaStream_t s) { cudaEventRecord(c->ev[2 * phase], s); }
static void toc(Ctx *c, int phase, cudaStream_t s) { cudaEventRecord(c->ev[2 * phase + 1], s); c->last_ms[phase] = 0.0; }

}  // namespace tkhp

using namespace tkhp;

// Every entry point runs with the context's device current and leaves the caller's current device
// as it found it (a process may hold contexts on several GPUs).
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        if (prev != dev) cudaSetDevice(dev); else prev = -1;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// Destroys whatever a (possibly half-built: zero-filled at birth) context owns besides the caller's workspace.
// The context's device is current.
static void release_ctx(Ctx *c) {
    for (int i = 0; i < 10; ++i) if (c->ev[i]) cudaEventDestroy(c->ev[i]);
    for (int i = 0; i < 2; ++i) if (c->copy_ev[i]) cudaEventDestroy(c->copy_ev[i]);
    for (int i = 0; i < 2; ++i) {
        if (c->side[i]) cudaStreamDestroy(c->side[i]);
        if (c->fork_ev[i]) cudaEventDestroy(c->fork_ev[i]);
        if (c->join_ev[i]) cudaEventDestroy(c->join_ev[i]);
    }
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    for (int w = 0; w < 3; ++w)
        for (int i = 0; i < 2 * PROF_MAX; ++i) if (c->prof_ev[w][i]) cudaEventDestroy(c->prof_ev[w][i]);
    for (int i = 0; i < Ctx::BUILD_GRAPH_SLOTS; ++i)
        if (c->build_slot[i].exec) cudaGraphExecDestroy(c->build_slot[i].exec);
    if (c->h_ring) cudaFreeHost(c->h_ring);
    if (c->h_scalars) cudaFreeHost(c->h_scalars);
    if (c->h_state) cudaFreeHost(c->h_state);
    cudaGetLastError();
    delete c;
}

extern "C" {

int tkhp_workspace_bytes(const tkhp_params *params, size_t *bytes) {
    char err[256];
    int rc = check_params(params, err, sizeof(err));
    if (rc) { snprintf(g_create_err, sizeof(g_create_err), "%s", err); return rc; }
    if (!bytes) return TKHP_EINVAL;
    *bytes = carve(nullptr, params, nullptr);
    return TKHP_OK;
}

int tkhp_create(const tkhp_params *params, void *d_workspace, size_t bytes, tkhp_ctx **out) {
    if (out) *out = nullptr;
    char err[256];
    int rc = check_params(params, err, sizeof(err));
    if (rc) { snprintf(g_create_err, sizeof(g_create_err), "%s", err); return rc; }
    if (!out || !d_workspace) { snprintf(g_create_err, sizeof(g_create_err), "NULL argument"); return TKHP_EINVAL; }
    if ((reinterpret_cast<uintptr_t>(d_workspace) & 255) != 0) { snprintf(g_create_err, sizeof(g_create_err), "workspace must be 256-byte aligned"); return TKHP_EINVAL; }
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev == 0 || params->device < 0 || params->device >= n_dev) {
        snprintf(g_create_err, sizeof(g_create_err), "no CUDA device %d (libtkhp has no CPU fallback)", params->device);
        cudaGetLastError();
        return TKHP_ECUDA;
    }
    DeviceGuard guard(params->device);      // the caller's current device comes back on every return path
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess || cur != params->device) { snprintf(g_create_err, sizeof(g_create_err), "cudaSetDevice failed"); cudaGetLastError(); return TKHP_ECUDA; }
    Ctx *c = new (std::nothrow) Ctx();
    if (!c) { snprintf(g_create_err, sizeof(g_create_err), "out of host memory"); return TKHP_EINVAL; }
    memset(c, 0, sizeof(Ctx));
    c->p = *params;
    // every failure below leaves through here: whatever was created so far is destroyed again
    auto fail = [&](int code, const char *msg) {
        snprintf(g_create_err, sizeof(g_create_err), "%s", msg);
        release_ctx(c);
        return code;
    };
    size_t need = carve(c, params, d_workspace);
    if (bytes < need) {
        char msg[128];
        snprintf(msg, sizeof(msg), "workspace too small: %zu < %zu bytes", bytes, need);
        return fail(TKHP_ECAPACITY, msg);
    }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, params->device) != cudaSuccess) return fail(TKHP_ECUDA, "cudaGetDeviceProperties failed");
    c->sm_count = prop.multiProcessorCount;
    atom_far_setup(c);
    c->fixed = params->precision == TKHP_FIXED;
    c->no_persist = (params->solver_flags & TKHP_SOLVER_NO_PERSISTENT) != 0;
    c->no_fused_step = (params->solver_flags & TKHP_SOLVER_NO_FUSED_STEP) != 0;
    c->test_barrier_fault = (params->solver_flags & TKHP_SOLVER_TEST_BARRIER_FAULT) != 0;
    if (cluster_pairs_configure(c) || atom_lists_configure(c) || atom_pairs_configure(c) || atom_solve_configure(c) || atom_stored_configure(c)) {
        char msg[sizeof(c->err)];
        snprintf(msg, sizeof(msg), "%s", c->err);
        return fail(TKHP_ECUDA, msg);
    }
    c->spec_iter = -1;
    c->fuse_q = false;
    c->n_noop_launches = 0;
    c->h_ring = c->d_ring = nullptr;
    if (cudaHostAlloc(&c->h_ring, RING * sizeof(double), cudaHostAllocMapped) != cudaSuccess ||
        cudaHostGetDevicePointer(&c->d_ring, c->h_ring, 0) != cudaSuccess ||
        cudaMallocHost(&c->h_scalars, 8 * sizeof(double)) != cudaSuccess ||
        cudaMallocHost(&c->h_state, sizeof(DeviceState)) != cudaSuccess)
        return fail(TKHP_ECUDA, "cudaMallocHost failed");
    bool ok = true;
    for (int i = 0; i < 10; ++i) ok &= cudaEventCreate(&c->ev[i]) == cudaSuccess;
    ok &= cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) == cudaSuccess;
    for (int i = 0; i < 2; ++i) ok &= cudaEventCreateWithFlags(&c->copy_ev[i], cudaEventDisableTiming) == cudaSuccess;
    for (int i = 0; i < 2; ++i) {
        ok &= cudaStreamCreateWithFlags(&c->side[i], cudaStreamNonBlocking) == cudaSuccess;
        ok &= cudaEventCreateWithFlags(&c->fork_ev[i], cudaEventDisableTiming) == cudaSuccess;
        ok &= cudaEventCreateWithFlags(&c->join_ev[i], cudaEventDisableTiming) == cudaSuccess;
    }
    for (int w = 0; w < 3; ++w)
        for (int i = 0; i < 2 * PROF_MAX; ++i) ok &= cudaEventCreate(&c->prof_ev[w][i]) == cudaSuccess;
    if (!ok) return fail(TKHP_ECUDA, "creating the context's streams and events failed");
    for (int i = 0; i < 5; ++i) c->last_ms[i] = -1.0;
    c->built = false;
    c->tstore_valid = false;
    c->header_valid = false;
    c->list_mode_in_use = TKHP_LIST_TILES;
    // the device-resident scalars start from zero (tickets, barrier words: tkhp_polar_energy may be the first call)
    if (cudaMemset(c->st, 0, sizeof(DeviceState)) != cudaSuccess || cluster_init(c) != TKHP_OK || cudaDeviceSynchronize() != cudaSuccess)
        return fail(TKHP_ECUDA, "initialising the workspace failed");
    *out = reinterpret_cast<tkhp_ctx *>(c);
    return TKHP_OK;
}

int tkhp_destroy(tkhp_ctx *ctx) {
    if (!ctx) return TKHP_EINVAL;
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    DeviceGuard guard(c->p.device);
    cudaDeviceSynchronize();
    release_ctx(c);
    return TKHP_OK;
}

const char *tkhp_last_error(const tkhp_ctx *ctx) {
    if (!ctx) return g_create_err;
    return reinterpret_cast<const Ctx *>(ctx)->err;
}

// everything tkhp_nblist_build enqueues: the prescribed block-pair list, then the finer lists
static int enqueue_build(Ctx *c, const double *d_pos, const double *d_polarizability, const int32_t *d_group_id,
                         cudaStream_t s) {
    int rc = nblist_build(c, d_pos, d_polarizability, d_group_id, s);
    if (rc == TKHP_OK && c->p.list_mode != TKHP_LIST_TILES) {
        rc = cluster_build(c, s);
        if (rc == TKHP_OK && c->p.list_mode == TKHP_LIST_ATOM) rc = atom_build(c, s);
    }
    const int rj = nblist_join(c, s);          // always: a forked branch must rejoin (stream capture)
    return rc ? rc : rj;
}

int tkhp_nblist_build(tkhp_ctx *ctx, const double *d_pos, const double *d_polarizability,
                      const int32_t *d_group_id, void *stream) {
    if (!ctx) return TKHP_EINVAL;
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    DeviceGuard guard(c->p.device);
    if (!d_pos || !d_polarizability || !d_group_id) return set_err(c, TKHP_EINVAL, "NULL input%s");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    tic(c, 0, s);
    c->header_valid = false;
    int rc = TKHP_OK;
    auto find_slot = [&]() {
        for (int i = 0; i < Ctx::BUILD_GRAPH_SLOTS; ++i) {
            const Ctx::BuildGraphSlot &g = c->build_slot[i];
            if (g.exec && g.key[0] == d_pos && g.key[1] == d_polarizability && g.key[2] == d_group_id) return i;
        }
        return -1;
    };
    // a caller who is capturing `s` into a graph of their own gets plain launches (they become nodes of that
    // graph); beginning a second capture on the stream would fail and replaying ours would nest it
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    const bool caller_capturing = s != nullptr && (cudaStreamIsCapturing(s, &cap) != cudaSuccess || cap != cudaStreamCaptureStatusNone);
    int slot = find_slot();
    if (slot < 0 && !c->no_graph && s != nullptr && !caller_capturing) {
        // capture the build once for these pointers (the legacy default stream cannot be captured) into the
        // least recently used slot
        int victim = 0;
        for (int i = 1; i < Ctx::BUILD_GRAPH_SLOTS; ++i)
            if (c->build_slot[i].used < c->build_slot[victim].used) victim = i;
        Ctx::BuildGraphSlot &g = c->build_slot[victim];
        if (g.exec) { cudaGraphExecDestroy(g.exec); g.exec = nullptr; }
        g.used = 0;
        cudaGraph_t graph = nullptr;
        const long long before = c->n_launches;
        if (cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
            rc = enqueue_build(c, d_pos, d_polarizability, d_group_id, s);
            const cudaError_t e = cudaStreamEndCapture(s, &graph);
            if (rc == TKHP_OK && e == cudaSuccess && graph && cudaGraphInstantiate(&g.exec, graph, 0) == cudaSuccess) {
                g.key[0] = d_pos; g.key[1] = d_polarizability; g.key[2] = d_group_id;
                g.launches = c->n_launches - before;
                c->n_graph_captures += 1;
                slot = victim;
            } else {
                g.exec = nullptr;
                c->no_graph = true;
                rc = TKHP_OK;
            }
            if (graph) cudaGraphDestroy(graph);
            c->n_launches = before;
        } else {
            c->no_graph = true;
        }
        cudaGetLastError();
    }
    if (slot >= 0 && !caller_capturing) {
        TKHP_CUDA(c, cudaGraphLaunch(c->build_slot[slot].exec, s));
        c->build_slot[slot].used = ++c->build_clock;
        c->n_launches += c->build_slot[slot].launches;
        c->n_graph_replays += 1;
    } else {
        rc = enqueue_build(c, d_pos, d_polarizability, d_group_id, s);
        if (rc) return rc;
        c->n_plain_builds += 1;
    }
    c->built = true;
    c->tstore_valid = false;               // stored matrix elements belong to the previous list
    c->list_mode_in_use = TKHP_LIST_TILES;
    toc(c, 0, s);
    return TKHP_OK;
}

int tkhp_nblist_view(tkhp_ctx *ctx, int32_t *n_blocks, int64_t *n_pairs, const int32_t **d_perm,
                     const int32_t **d_pairs, void *stream) {
    if (!ctx) return TKHP_EINVAL;
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    DeviceGuard guard(c->p.device);
    int rc = ensure_header(c, static_cast<cudaStream_t>(stream));
    if (rc) return rc;
    if (n_blocks) *n_blocks = c->n_blocks;
    if (n_pairs) *n_pairs = c->n_tiles_host;
    if (d_perm) *d_perm = c->perm;
    if (d_pairs) *d_pairs = reinterpret_cast<const int32_t *>(c->pairs);
    return TKHP_OK;
}

int tkhp_nblist_stats(tkhp_ctx *ctx, int64_t *n_pairs_within_cutoff, int64_t *n_slots_evaluated,
                      int32_t *list_mode_in_use, void *stream) {
    if (!ctx) return TKHP_EINVAL;
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    DeviceGuard guard(c->p.device);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int rc = ensure_header(c, s);
    if (rc) return rc;
    if (n_pairs_within_cutoff) {
        rc = nblist_count_pairs(c, s);
        if (rc) return rc;
        TKHP_CUDA(c, cudaMemcpyAsync(c->h_scalars, &c->st->n_pairs_within_cutoff, sizeof(long long), cudaMemcpyDeviceToHost, s));
        TKHP_CUDA(c, cudaStreamSynchronize(s));
        long long v;
        memcpy(&v, c->h_scalars, sizeof(v));
        *n_pairs_within_cutoff = v;
    }
    if (n_slots_evaluated) {
        if (c->list_mode_in_use == TKHP_LIST_ATOM) {
            *n_slots_evaluated = atom_slots(c);
        } else if (c->list_mode_in_use == TKHP_LIST_CLUSTER) {
            *n_slots_evaluated = cluster_slots(c);
        } else {
            const long long diag = c->n_blocks;
            *n_slots_evaluated = (c->n_tiles_host - diag) * 1024 + diag * 992;
        }
    }
    if (list_mode_in_use) *list_mode_in_use = c->list_mode_in_use;
    return TKHP_OK;
}

int tkhp_nblist_atom_stats(tkhp_ctx *ctx, int64_t out[4], void *stream) {
    if (!ctx || !out) return TKHP_EINVAL;
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    DeviceGuard guard(c->p.device);
    int rc = ensure_header(c, static_cast<cudaStream_t>(stream));
    if (rc) return rc;
    out[0] = out[1] = out[2] = out[3] = 0;
    if (c->list_mode_in_use != TKHP_LIST_ATOM) return TKHP_OK;
    const DeviceState &h = *c->h_state;
    out[0] = 32LL * h.n_atom_far;
    out[1] = 32LL * (h.n_atom_entries - h.n_atom_far);
    out[2] = h.n_atom_segments;
    out[3] = c->far_on ? 1 : 0;
    return TKHP_OK;
}

int tkhp_perm_field(tkhp_ctx *ctx, const double *d_charge, const double *d_dipole, const double *d_quad,
                    double *d_field, void *stream) {
    if (!ctx) return TKHP_EINVAL;
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    DeviceGuard guard(c->p.device);
    if (!d_charge || !d_dipole || !d_quad || !d_field) return set_err(c, TKHP_EINVAL, "NULL argument%s");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int rc = ensure_header(c, s);
    if (rc) return rc;
    tic(c, 1, s);
    rc = do_perm_field(c, d_charge, d_dipole, d_quad, d_field, s);
    toc(c, 1, s);
    return rc;
}

int tkhp_tmatvec(tkhp_ctx *ctx, const double *d_mu, double *d_out, void *stream) {
    if (!ctx) return TKHP_EINVAL;
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    DeviceGuard guard(c->p.device);
    if (!d_mu || !d_out || d_mu == d_out) return set_err(c, TKHP_EINVAL, "NULL or aliased argument%s");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int rc = ensure_header(c, s);
    if (rc) return rc;
    tic(c, 2, s);
    rc = do_tmatvec(c, d_mu, d_out, s);
    toc(c, 2, s);
    return rc;
}

int tkhp_polar_solve(tkhp_ctx *ctx, const double *d_field, double *d_mu, double tol, int32_t max_iter,
                     int32_t use_guess, int32_t *h_iters, double *h_rms, void *stream) {
    if (!ctx) return TKHP_EINVAL;
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    DeviceGuard guard(c->p.device);
    if (!d_field || !d_mu || !(tol > 0.0) || max_iter < 0) return set_err(c, TKHP_EINVAL, "bad argument%s");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int rc = ensure_header(c, s);
    if (rc) return rc;
    tic(c, 3, s);
    rc = do_polar_solve(c, d_field, d_mu, tol, max_iter, use_guess, h_iters, h_rms, s);
    toc(c, 3, s);
    return rc;
}

int tkhp_polar_energy(tkhp_ctx *ctx, const double *d_mu, const double *d_field, double *d_energy, void *stream) {
    if (!ctx) return TKHP_EINVAL;
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    DeviceGuard guard(c->p.device);
    if (!d_mu || !d_field || !d_energy) return set_err(c, TKHP_EINVAL, "NULL argument%s");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    tic(c, 4, s);
    int rc = do_polar_energy(c, d_mu, d_field, d_energy, s);
    toc(c, 4, s);
    return rc;
}

int tkhp_polarize_host(tkhp_ctx *ctx, const double *h_pos, const double *h_polarizability,
                       const int32_t *h_group_id, const double *h_charge, const double *h_dipole,
                       const double *h_quad, double tol, int32_t max_iter, double *h_mu, double *h_field,
                       double *h_energy, int32_t *h_iters, double *h_rms, void *stream) {
    if (!ctx) return TKHP_EINVAL;
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    DeviceGuard guard(c->p.device);
    if (!h_pos || !h_polarizability || !h_group_id || !h_charge || !h_dipole || !h_quad || !h_energy)
        return set_err(c, TKHP_EINVAL, "NULL argument%s");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const size_t n = c->n;
    TKHP_CUDA(c, cudaMemcpyAsync(c->h_pos, h_pos, 24 * n, cudaMemcpyHostToDevice, s));
    TKHP_CUDA(c, cudaMemcpyAsync(c->h_alpha, h_polarizability, 8 * n, cudaMemcpyHostToDevice, s));
    TKHP_CUDA(c, cudaMemcpyAsync(c->h_group, h_group_id, 4 * n, cudaMemcpyHostToDevice, s));
    // the multipoles (80 of the 116 bytes per atom) are not needed before the field: their copies
    // run on a second stream beside the list build (copy engine and SMs at the same time)
    TKHP_CUDA(c, cudaEventRecord(c->copy_ev[0], s));               // after whatever the caller queued on s
    TKHP_CUDA(c, cudaStreamWaitEvent(c->copy_stream, c->copy_ev[0], 0));
    TKHP_CUDA(c, cudaMemcpyAsync(c->h_charge, h_charge, 8 * n, cudaMemcpyHostToDevice, c->copy_stream));
    TKHP_CUDA(c, cudaMemcpyAsync(c->h_dipole, h_dipole, 24 * n, cudaMemcpyHostToDevice, c->copy_stream));
    TKHP_CUDA(c, cudaMemcpyAsync(c->h_quad, h_quad, 48 * n, cudaMemcpyHostToDevice, c->copy_stream));
    TKHP_CUDA(c, cudaEventRecord(c->copy_ev[1], c->copy_stream));
    int rc = tkhp_nblist_build(ctx, c->h_pos, c->h_alpha, c->h_group, stream);
    if (rc) { cudaStreamSynchronize(c->copy_stream); return rc; }
    TKHP_CUDA(c, cudaStreamWaitEvent(s, c->copy_ev[1], 0));
    rc = tkhp_perm_field(ctx, c->h_charge, c->h_dipole, c->h_quad, c->h_field, stream);
    if (rc) { cudaStreamSynchronize(c->copy_stream); return rc; }     // the caller may free its buffers
    int rc_solve = tkhp_polar_solve(ctx, c->h_field, c->h_mu, tol, max_iter, 0, h_iters, h_rms, stream);
    if (rc_solve && rc_solve != TKHP_ENOCONV) return rc_solve;
    rc = tkhp_polar_energy(ctx, c->h_mu, c->h_field, c->h_energy, stream);
    if (rc) return rc;
    if (h_mu) TKHP_CUDA(c, cudaMemcpyAsync(h_mu, c->h_mu, 24 * n, cudaMemcpyDeviceToHost, s));
    if (h_field) TKHP_CUDA(c, cudaMemcpyAsync(h_field, c->h_field, 24 * n, cudaMemcpyDeviceToHost, s));
    TKHP_CUDA(c, cudaMemcpyAsync(h_energy, c->h_energy, 8, cudaMemcpyDeviceToHost, s));
    TKHP_CUDA(c, cudaStreamSynchronize(s));
    return rc_solve;
}

int tkhp_profile_reset(tkhp_ctx *ctx, int32_t enable_kernel_events) {
    if (!ctx) return TKHP_EINVAL;
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    DeviceGuard guard(c->p.device);
    c->n_launches = 0;
    c->n_noop_launches = 0;
    c->prof = enable_kernel_events != 0;
    c->prof_n[0] = c->prof_n[1] = c->prof_n[2] = 0;
    c->prof_solve_matvecs = 0;
    return TKHP_OK;
}

int tkhp_profile_read(tkhp_ctx *ctx, int64_t *n_kernel_launches, int32_t *n_tmatvec_kernels,
                      double *tmatvec_kernel_ms, int32_t *n_field_kernels, double *field_kernel_ms) {
    if (!ctx) return TKHP_EINVAL;
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    DeviceGuard guard(c->p.device);
    if (n_kernel_launches) *n_kernel_launches = c->n_launches - c->n_noop_launches;
    double tot[2] = {0.0, 0.0};
    int cnt[2] = {0, 0};
    for (int w = 0; w < 2; ++w) {
        for (int i = 0; i < c->prof_n[w]; ++i) {
            if (c->prof_skip[w][i]) continue;
            float t = 0.f;
            if (cudaEventSynchronize(c->prof_ev[w][2 * i + 1]) != cudaSuccess ||
                cudaEventElapsedTime(&t, c->prof_ev[w][2 * i], c->prof_ev[w][2 * i + 1]) != cudaSuccess) {
                cudaGetLastError();
                return set_err(c, TKHP_ECUDA, "profile events not complete%s");
            }
            tot[w] += t;
            cnt[w]++;
        }
    }
    if (n_tmatvec_kernels) *n_tmatvec_kernels = cnt[0];
    if (tmatvec_kernel_ms) *tmatvec_kernel_ms = tot[0];
    if (n_field_kernels) *n_field_kernels = cnt[1];
    if (field_kernel_ms) *field_kernel_ms = tot[1];
    return TKHP_OK;
}

int tkhp_profile_read_solve(tkhp_ctx *ctx, int32_t *n_solve_kernels, double *solve_kernel_ms, int64_t *n_matvecs) {
    if (!ctx) return TKHP_EINVAL;
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    DeviceGuard guard(c->p.device);
    double tot = 0.0;
    for (int i = 0; i < c->prof_n[2]; ++i) {
        float t = 0.f;
        if (cudaEventSynchronize(c->prof_ev[2][2 * i + 1]) != cudaSuccess ||
            cudaEventElapsedTime(&t, c->prof_ev[2][2 * i], c->prof_ev[2][2 * i + 1]) != cudaSuccess) {
            cudaGetLastError();
            return set_err(c, TKHP_ECUDA, "profile events not complete%s");
        }
        tot += t;
    }
    if (n_solve_kernels) *n_solve_kernels = c->prof_n[2];
    if (solve_kernel_ms) *solve_kernel_ms = tot;
    if (n_matvecs) *n_matvecs = c->prof_solve_matvecs;
    return TKHP_OK;
}

int tkhp_profile_read_build(tkhp_ctx *ctx, int64_t out[5]) {
    if (!ctx || !out) return TKHP_EINVAL;
    const Ctx *c = reinterpret_cast<const Ctx *>(ctx);
    out[0] = c->n_graph_captures;
    out[1] = c->n_graph_replays;
    out[2] = c->n_plain_builds;
    out[3] = c->no_graph ? 1 : 0;
    out[4] = c->n_barrier_timeouts;
    return TKHP_OK;
}

int tkhp_last_timings(tkhp_ctx *ctx, double ms[5]) {
    if (!ctx || !ms) return TKHP_EINVAL;
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    DeviceGuard guard(c->p.device);
    for (int ph = 0; ph < 5; ++ph) {
        if (c->last_ms[ph] < 0.0) { ms[ph] = -1.0; continue; }
        float t = 0.f;
        if (cudaEventSynchronize(c->ev[2 * ph + 1]) != cudaSuccess ||
            cudaEventElapsedTime(&t, c->ev[2 * ph], c->ev[2 * ph + 1]) != cudaSuccess) {
            cudaGetLastError();
            ms[ph] = -1.0;
            continue;
        }
        ms[ph] = t;
    }
    return TKHP_OK;
}

}  // extern "C"

// api.cu -- the C ABI of include/petar.h: argument checks, workspace carving, launch sequences.
#include <stdio.h>
#include <string.h>
#include <stdlib.h>
#include <atomic>
#include <new>
#include "internal.cuh"

static thread_local cudaError_t g_last_cuda = cudaSuccess;
static std::atomic<long long> g_launches{0};
static int g_profiling = 0;

void petar_count_launch(int n) { g_launches += n; }
void petar_debug_check(cudaStream_t s, const char* name) {
    static int mode = -1;
    if (mode < 0) { const char* e = getenv("PETAR_DEBUG_SYNC"); mode = (e && e[0] == '1') ? 1 : 0; }
    if (!mode) return;
    cudaError_t e = cudaStreamSynchronize(s);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) fprintf(stderr, "[petar] kernel %s failed: %s\n", name, cudaGetErrorString(e));
}
// Stage timing: events are only RECORDED here (asynchronously, on the caller's stream);
// petar_stage_times synchronises on them later.  No effect unless petar_set_profiling(1)
// was called before petar_tree_build.
void stage_begin(petar_tree* t, int stage, cudaStream_t s) {
    if (!t->ev) return;
    cudaEventRecord(t->ev[2 * stage], s);
}
void stage_end(petar_tree* t, int stage, cudaStream_t s) {
    if (!t->ev) return;
    cudaEventRecord(t->ev[2 * stage + 1], s);
    t->stage_rec[stage] = 1;
}

#define CK(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { g_last_cuda = e_; return PETAR_ECUDA; } } while (0)

static inline size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

static bool params_ok(const petar_params* p) {
    if (!p) return false;
    if (!(p->G == p->G) || !(p->theta >= 0.0) || !(p->r_in_over_r_out > 0.0 && p->r_in_over_r_out < 1.0)) return false;
    if (p->multipole != 1 && p->multipole != 2) return false;
    if (p->n_leaf_limit < 1 || p->n_leaf_limit > 64) return false;
    if (p->n_group_limit < p->n_leaf_limit || p->n_group_limit > 64) return false;
    if (p->flags != 0) return false;
    if (!(p->list_entries_per_particle == p->list_entries_per_particle) || !(p->nodes_per_particle == p->nodes_per_particle)) return false;
    return true;
}

// default: N + 4096 nodes for n_leaf_limit >= 4, else 3N + 4096 (measured: 0.35 N at config 3 with leaves of 8).  Rule O5 keeps
// single-child chains, so no multiple of N is a hard bound (a tight binary deep in the tree adds a node per level):
// nodes_per_particle raises the capacity, PETAR_ST_NODE_CAP reports an overflow.
static int node_capacity(int64_t N, const petar_params* p) {
    double per = p->nodes_per_particle > 0.0 ? p->nodes_per_particle : (p->n_leaf_limit >= 4 ? 1.0 : 3.0);
    double cap = per * (double)N + 4096.0;
    if (cap > 2.0e9) cap = 2.0e9;
    return (int)cap;
}
static long long arena_chunks_for(int64_t N, const petar_params* p) {
    double per = p->list_entries_per_particle > 0.0 ? p->list_entries_per_particle : 1024.0;
    double entries = per * (double)N;
    if (p->list_entries_per_particle <= 0.0 && entries < 16.0 * 1024 * 1024) entries = 16.0 * 1024 * 1024;
    long long chunks = (long long)(entries / PETAR_CHUNK) + 64;
    if (chunks > 2000000000ll / 1) chunks = 2000000000ll;
    return chunks;
}

// Carves the workspace; with base == nullptr only sizes it.
static size_t carve(Workspace* w, char* base, int64_t N, const petar_params* p) {
    size_t off = 0;
    auto take = [&](size_t bytes) -> char* { char* r = base ? base + off : nullptr; off += align_up(bytes); return r; };
    const size_t n = (size_t)N;
    const int nblk = (int)((N + 2047) / 2048) + 1;
    const int ntile = (int)((N + 1023) / 1024) + 1;
    Workspace tmp; Workspace* W = w ? w : &tmp;
    W->hdr = (DevHeader*)take(sizeof(DevHeader));
    W->key = (unsigned long long*)take(n * 8); W->key_alt = (unsigned long long*)take(n * 8);
    W->idx = (unsigned*)take(n * 4); W->idx_alt = (unsigned*)take(n * 4);
    W->sort_hist = (unsigned*)take(8 * 256 * 4);
    W->sort_blk = (unsigned*)take((size_t)256 * nblk * 4);
    W->rec = (double2*)take(n * 64);
    W->xs = (double*)take(n * 8); W->ys = (double*)take(n * 8); W->zs = (double*)take(n * 8);
    W->ms = (double*)take(n * 8); W->routs = (double*)take(n * 8); W->rss = (double*)take(n * 8);
    W->vxs = (double*)take(n * 8); W->vys = (double*)take(n * 8); W->vzs = (double*)take(n * 8);
    W->pa = (float4*)take(n * 16); W->pb = (float4*)take(n * 16);
    W->D = (signed char*)take(n + 1); W->depth = (signed char*)take(n); W->glevel = (signed char*)take(n);
    W->gflag = (int*)take((2 * (n + 1)) * 4);
    W->tile_cnt = (int*)take((size_t)PETAR_NLEVELS * ntile * 4);
    W->scan_tmp = (int*)take((size_t)(3 * (n + 1) / 4096 + 8) * 8);     // partials of the longest scan (3 entries per group, list export)
    W->node_cap = node_capacity(N, p);
    W->nint = (NodeInt*)take((size_t)W->node_cap * sizeof(NodeInt));
    W->nmac = (NodeMac*)take((size_t)W->node_cap * sizeof(NodeMac));
    W->nmom = (NodeMom*)take((size_t)W->node_cap * sizeof(NodeMom));
    W->nsp = (NodeSp*)take((size_t)W->node_cap * sizeof(NodeSp));
    W->nw = (NodeW*)take((size_t)W->node_cap * sizeof(NodeW));
    W->group_cap = (int)N + 1;
    W->grp = (GroupRec*)take((size_t)W->group_cap * sizeof(GroupRec));
    W->srec = (SuperRec*)take((size_t)PETAR_NSUP * W->group_cap * sizeof(SuperRec));
    W->smap = (int*)take((size_t)PETAR_NSUP * n * 4);
    W->unit_cap = (int)(PETAR_NSUP * (N + 64));             // every unit holds at least one particle
    W->units = (ForceUnit*)take((size_t)W->unit_cap * sizeof(ForceUnit));
    W->part = (double*)take((size_t)(PETAR_NSUP + 1) * n * 4 * 8);
    W->part_s = (double*)take((size_t)(PETAR_NSUP + 1) * n * 8);
    W->refine_q = (int*)take(n * 2 * 4);
    W->nb_cnt = (int*)take(n * 4);
    W->nb_queue = (int*)take(((size_t)W->group_cap + 1) * 4);
    W->exp_scratch = (int*)take((10 * (n + 1) + 8) * 4);
    long long chunks = arena_chunks_for(N, p);
    W->arena_chunks = (int)chunks;
    W->arena = (int*)take((size_t)chunks * PETAR_CHUNK * 4);
    return off;
}

extern "C" size_t petar_workspace_bytes(int64_t N, const petar_params* p) {
    if (N < 0 || N > 2000000000ll || !params_ok(p)) return 0;
    return carve(nullptr, nullptr, N, p) + 256;
}

static void free_handle(petar_tree* t) {
    if (t->ev) { for (int k = 0; k < 2 * PETAR_N_STAGES; ++k) if (t->ev[k]) cudaEventDestroy(t->ev[k]); delete[] t->ev; }
    if (t->ev_fork) cudaEventDestroy(t->ev_fork);
    if (t->ev_join) cudaEventDestroy(t->ev_join);
    if (t->ev_tab) cudaEventDestroy(t->ev_tab);
    if (t->side) cudaStreamDestroy(t->side);
    t->magic = 0;
    delete t;
}

// S0-S6 into the handle's workspace (shared by petar_tree_build and petar_tree_rebuild)
static int build_into(petar_tree* t, const double* x, const double* y, const double* z, const double* m, const double* r_out,
                      const double* r_search, cudaStream_t s) {
    t->x = x; t->y = y; t->z = z; t->m = m; t->r_out = r_out; t->r_search = r_search;
    t->built = false; t->walked = false; t->nb_counted = false;
    for (int k = 0; k < PETAR_N_STAGES; ++k) t->stage_rec[k] = 0;
    if (g_profiling && !t->ev) {            // events are created once per handle, never on a rebuild
        t->ev = new (std::nothrow) cudaEvent_t[2 * PETAR_N_STAGES];
        if (!t->ev) return PETAR_EINVAL;
        for (int k = 0; k < 2 * PETAR_N_STAGES; ++k) t->ev[k] = nullptr;
        for (int k = 0; k < 2 * PETAR_N_STAGES; ++k) CK(cudaEventCreate(&t->ev[k]));
    }
    if (!t->side) {                         // once per handle
        CK(cudaStreamCreateWithFlags(&t->side, cudaStreamNonBlocking));
        CK(cudaEventCreateWithFlags(&t->ev_fork, cudaEventDisableTiming));
        CK(cudaEventCreateWithFlags(&t->ev_join, cudaEventDisableTiming));
        CK(cudaEventCreateWithFlags(&t->ev_tab, cudaEventDisableTiming));
    }
    if (t->N > 0) {
        CK(launch_keys_sort_gather(t, s));
        CK(launch_tree(t, s));
    }
    t->built = true;
    return PETAR_OK;
}

extern "C" int petar_tree_build(const double* x, const double* y, const double* z, const double* m, const double* r_out,
                                const double* r_search, int64_t N, const petar_params* p, void* workspace,
                                size_t workspace_bytes, void* cuda_stream, petar_tree** tree_out) {
    if (!tree_out) return PETAR_EINVAL;
    *tree_out = nullptr;
    if (N < 0 || N > 2000000000ll || !params_ok(p)) return PETAR_EINVAL;
    if (N > 0 && (!x || !y || !z || !m || !r_out)) return PETAR_EINVAL;
    size_t need = petar_workspace_bytes(N, p);
    if (N > 0 && (!workspace || workspace_bytes < need || ((uintptr_t)workspace & 255u))) return PETAR_EWORKSPACE;
    petar_tree* t = new (std::nothrow) petar_tree();
    if (!t) return PETAR_EINVAL;
    memset(t, 0, sizeof(*t));
    t->magic = PETAR_MAGIC; t->N = N; t->p = *p;
    t->workspace = workspace; t->workspace_bytes = workspace_bytes;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&t->sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) { g_last_cuda = e; free_handle(t); return PETAR_ECUDA; }
    if (N > 0) carve(&t->w, (char*)workspace, N, p);
    int rc = build_into(t, x, y, z, m, r_out, r_search, (cudaStream_t)cuda_stream);
    if (rc) { free_handle(t); return rc; }
    *tree_out = t;
    return PETAR_OK;
}

extern "C" int petar_tree_rebuild(petar_tree* t, const double* x, const double* y, const double* z, const double* m,
                                  const double* r_out, const double* r_search, void* cuda_stream) {
    if (!t || t->magic != PETAR_MAGIC) return PETAR_ENOTBUILT;
    if (t->N > 0 && (!x || !y || !z || !m || !r_out)) return PETAR_EINVAL;
    return build_into(t, x, y, z, m, r_out, r_search, (cudaStream_t)cuda_stream);
}

#define OVERLAP_WALK_CTAS 2      // CTAs per SM of k_walk / k_force_units while the two run side by side
static int check_tree(petar_tree* t) { return (t && t->magic == PETAR_MAGIC && t->built) ? PETAR_OK : PETAR_ENOTBUILT; }

static int ensure_walk(petar_tree* t, cudaStream_t s) {
    if (t->walked) return PETAR_OK;
    CK(launch_walk(t, s));
    t->walked = true;
    return PETAR_OK;
}

// reads the device header into *out (HOST) and synchronises
static int read_header(petar_tree* t, cudaStream_t s, DevHeader* out) {
    CK(cudaMemcpyAsync(out, t->w.hdr, sizeof(DevHeader), cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    return PETAR_OK;
}

extern "C" int petar_long_range_force(petar_tree* t, double* acc_x, double* acc_y, double* acc_z, double* pot,
                                      petar_counts* counts, void* cuda_stream) {
    int rc = check_tree(t);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (t->N == 0) { if (counts) memset(counts, 0, sizeof(*counts)); return PETAR_OK; }
    if (!t->walked) {
        // Force phase A needs the super-group walks only.  The per-group walk (latency- and integer-bound) runs beside it on
        // the handle's second stream: phase A is bound by the FMA pipe and leaves half of the issue slots free.
        CK(launch_walk_supers(t, s));
        CK(cudaEventRecord(t->ev_fork, s));
        CK(cudaStreamWaitEvent(t->side, t->ev_fork, 0));
        // From here on the side stream may hold work that uses the workspace: whatever fails, the caller's stream is made to
        // wait for it before this call returns, so that an error return never leaves work running behind the caller's back.
        cudaError_t fe = [&]() -> cudaError_t {
            cudaError_t e;
            if ((e = launch_walk_groups(t, t->side, OVERLAP_WALK_CTAS)) != cudaSuccess) return e;   // launched first: its CTAs take their place on the SMs before the unit kernels'
            if ((e = launch_force_units_table(t, s)) != cudaSuccess) return e;
            if ((e = cudaEventRecord(t->ev_tab, s)) != cudaSuccess) return e;
            if ((e = launch_force_units_tc(t, s)) != cudaSuccess) return e;
            if ((e = cudaStreamWaitEvent(t->side, t->ev_tab, 0)) != cudaSuccess) return e;
            if ((e = launch_force_units_small(t, t->side)) != cudaSuccess) return e;   // the small units and the changeover pairs follow the walk on the side
            return launch_force_near(t, t->side);                                      // stream, beside the tail of the tensor-core kernel
        }();
        cudaError_t je = cudaEventRecord(t->ev_join, t->side);
        if (je == cudaSuccess) je = cudaStreamWaitEvent(s, t->ev_join, 0);
        if (je != cudaSuccess) cudaStreamSynchronize(t->side);      // could not order the streams on the device: wait on the host instead
        CK(fe);
        CK(je);
        stage_end(t, PETAR_STAGE_FORCE_UNITS, s);
        t->walked = true;
        CK(launch_force_groups(t, acc_x, acc_y, acc_z, pot, s));
    } else {
        CK(launch_force(t, acc_x, acc_y, acc_z, pot, s));
    }
    if (counts) {
        DevHeader hh;
        rc = read_header(t, s, &hh);
        if (rc) return rc;
        counts->n_groups = hh.n_groups; counts->n_nodes = hh.n_nodes;
        counts->n_epep = (int64_t)hh.n_epep; counts->n_epsp = (int64_t)hh.n_epsp; counts->n_epep_near = (int64_t)hh.n_epep_near;
        counts->n_ep_list = (int64_t)hh.n_ep_list; counts->n_sp_list = (int64_t)hh.n_sp_list;
        counts->list_entries_used = (int64_t)hh.arena_top * PETAR_CHUNK;
        counts->n_epsp_common = (int64_t)hh.n_epsp_common;
        counts->n_refined = (int64_t)hh.n_refine;
        if (hh.status & PETAR_ST_FATAL) return PETAR_ESTATUS;      // the bits that made the kernels write nothing
    }
    return PETAR_OK;
}

extern "C" int petar_neighbor_list(petar_tree* t, int64_t* offsets, int32_t* indices, int64_t capacity, int32_t* status_dev,
                                   void* cuda_stream) {
    int rc = check_tree(t);
    if (rc) return rc;
    if (!offsets || capacity < 0) return PETAR_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (t->N == 0) {
        CK(cudaMemsetAsync(offsets, 0, 8, s));
        if (status_dev) CK(cudaMemsetAsync(status_dev, 0, 4, s));
        return PETAR_OK;
    }
    rc = ensure_walk(t, s);
    if (rc) return rc;
    CK(launch_neighbors(t, offsets, indices, capacity, status_dev, s));
    return PETAR_OK;
}

extern "C" int petar_search_radii(const double* vx, const double* vy, const double* vz, const double* r_out, double C_r, double dt_L,
                                  int64_t N, double* r_search_out, void* cuda_stream) {
    if (N < 0 || !(C_r >= 0.0) || !(dt_L >= 0.0)) return PETAR_EINVAL;
    if (N == 0) return PETAR_OK;
    if (!vx || !vy || !vz || !r_out || !r_search_out) return PETAR_EINVAL;
    CK(launch_search_radii(vx, vy, vz, r_out, C_r, dt_L, N, r_search_out, (cudaStream_t)cuda_stream));
    return PETAR_OK;
}

extern "C" int petar_neighbor_list_orbit(petar_tree* t, const double* vx, const double* vy, const double* vz, double C_V,
                                         int64_t* offsets, int32_t* indices, int64_t capacity, int32_t* status_dev, void* cuda_stream) {
    int rc = check_tree(t);
    if (rc) return rc;
    if (!offsets || capacity < 0 || !(C_V >= 0.0)) return PETAR_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (t->N == 0) {
        CK(cudaMemsetAsync(offsets, 0, 8, s));
        if (status_dev) CK(cudaMemsetAsync(status_dev, 0, 4, s));
        return PETAR_OK;
    }
    if (!vx || !vy || !vz) return PETAR_EINVAL;
    rc = ensure_walk(t, s);
    if (rc) return rc;
    CK(launch_neighbors(t, offsets, indices, capacity, status_dev, s, vx, vy, vz, C_V));
    return PETAR_OK;
}

extern "C" size_t petar_clusters_workspace_bytes(int64_t N) { return N < 0 ? 0 : clusters_workspace_bytes(N); }

extern "C" int petar_clusters(const int64_t* offsets, const int32_t* indices, int64_t N, int32_t* label, int64_t* n_clusters_dev,
                              int64_t* cluster_offsets, int32_t* members, void* workspace, size_t workspace_bytes, void* cuda_stream) {
    if (N < 0 || N > 2000000000ll) return PETAR_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (N == 0) {
        if (n_clusters_dev) CK(cudaMemsetAsync(n_clusters_dev, 0, 8, s));
        if (cluster_offsets) CK(cudaMemsetAsync(cluster_offsets, 0, 8, s));
        return PETAR_OK;
    }
    if (!offsets || !label) return PETAR_EINVAL;
    if (members && !cluster_offsets) return PETAR_EINVAL;
    if (cluster_offsets && (!workspace || workspace_bytes < clusters_workspace_bytes(N) || ((uintptr_t)workspace & 255u))) return PETAR_EWORKSPACE;
    CK(launch_clusters((const long long*)offsets, indices, N, label, (long long*)n_clusters_dev, (long long*)cluster_offsets, members, workspace, s));
    return PETAR_OK;
}

extern "C" int petar_tree_status(petar_tree* t, int32_t* status_host, void* cuda_stream) {
    int rc = check_tree(t);
    if (rc) return rc;
    if (!status_host) return PETAR_EINVAL;
    if (t->N == 0) { *status_host = 0; return PETAR_OK; }
    DevHeader hh;
    rc = read_header(t, (cudaStream_t)cuda_stream, &hh);
    if (rc) return rc;
    *status_host = hh.status;
    return PETAR_OK;
}

extern "C" int petar_tree_destroy(petar_tree* t) {
    if (!t) return PETAR_OK;
    if (t->magic != PETAR_MAGIC) return PETAR_ENOTBUILT;
    free_handle(t);
    return PETAR_OK;
}

extern "C" const char* petar_strerror(int code) {
    switch (code) {
        case PETAR_OK: return "ok";
        case PETAR_EINVAL: return "invalid argument";
        case PETAR_EWORKSPACE: return "workspace too small or misaligned";
        case PETAR_ECUDA: return cudaGetErrorString(g_last_cuda);
        case PETAR_ENOTBUILT: return "no tree built / handle destroyed";
        case PETAR_ESTATUS: return "device status word non-zero (see petar_tree_status)";
        case PETAR_ECAPACITY: return "N exceeds the fixed capacity of the library's built-in scratch array (PETAR_SHORT_RANGE_NOALLOC_MAX_N); use the call that takes a workspace";
        default: return "unknown error";
    }
}

extern "C" int petar_debug_export(petar_tree* t, int what, void* dst, size_t dst_bytes, void* cuda_stream) {
    int rc = check_tree(t);
    if (rc) return rc;
    if (!dst) return PETAR_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (t->N == 0) return PETAR_OK;
    DevHeader hh;
    rc = read_header(t, s, &hh);
    if (rc) return rc;
    t->h_nodes = hh.n_nodes; t->h_groups = hh.n_groups;
    const size_t n = (size_t)t->N;
    const Workspace& w = t->w;
    auto copy = [&](const void* src, size_t bytes) -> int {
        if (dst_bytes < bytes) return PETAR_EINVAL;
        CK(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, s));
        return PETAR_OK;
    };
    switch (what) {
        case PETAR_DBG_HEADER: {
            long long v[8] = {hh.n_nodes, hh.n_groups, hh.status, (long long)hh.arena_top * PETAR_CHUNK, 0, 0, 0, 0};
            if (dst_bytes < sizeof(v)) return PETAR_EINVAL;
            CK(cudaMemcpyAsync(dst, v, sizeof(v), cudaMemcpyHostToDevice, s));
            break;
        }
        case PETAR_DBG_ROOT: {
            double v[4] = {hh.c[0], hh.c[1], hh.c[2], hh.h};
            if (dst_bytes < sizeof(v)) return PETAR_EINVAL;
            CK(cudaMemcpyAsync(dst, v, sizeof(v), cudaMemcpyHostToDevice, s));
            break;
        }
        case PETAR_DBG_KEYS: rc = copy(w.key, n * 8); break;
        case PETAR_DBG_PERM: rc = copy(w.idx, n * 4); break;
        case PETAR_DBG_NODE_INT: rc = copy(w.nint, (size_t)hh.n_nodes * sizeof(NodeInt)); break;
        case PETAR_DBG_NODE_DBL: case PETAR_DBG_GROUP_INT: case PETAR_DBG_GROUP_DBL: case PETAR_DBG_GROUP_CNT: case PETAR_DBG_GROUP_SUPER:
        case PETAR_DBG_LIST_OFFS: case PETAR_DBG_LISTS: {
            if ((what == PETAR_DBG_GROUP_CNT || what == PETAR_DBG_GROUP_SUPER || what == PETAR_DBG_LIST_OFFS || what == PETAR_DBG_LISTS) && !t->walked) return PETAR_ENOTBUILT;
            cudaError_t e = launch_export_lists(t, what, dst, dst_bytes, s);
            if (e == cudaErrorInvalidValue) return PETAR_EINVAL;
            CK(e);
            break;
        }
        default: return PETAR_EINVAL;
    }
    if (rc) return rc;
    CK(cudaStreamSynchronize(s));
    return PETAR_OK;
}

extern "C" int petar_set_profiling(int on) { g_profiling = on ? 1 : 0; return PETAR_OK; }
extern "C" int petar_stage_times(petar_tree* t, float* stage_ms) {
    int rc = check_tree(t);
    if (rc) return rc;
    if (!stage_ms) return PETAR_EINVAL;
    for (int k = 0; k < PETAR_N_STAGES; ++k) {
        stage_ms[k] = 0.f;
        if (t->ev && t->stage_rec[k]) {
            CK(cudaEventSynchronize(t->ev[2 * k + 1]));
            CK(cudaEventElapsedTime(&stage_ms[k], t->ev[2 * k], t->ev[2 * k + 1]));
        }
    }
    return PETAR_OK;
}
extern "C" int64_t petar_launch_count(void) { return (int64_t)g_launches.load(); }

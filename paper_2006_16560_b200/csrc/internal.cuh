// internal.cuh -- shared declarations of the CUDA path (host handle, HBM layout, launch wrappers).
// Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/petar.h"
// status bits that leave the tree or its interaction lists unusable: the force kernels write nothing when one is set.
// PETAR_ST_NB_CAP is not among them -- a neighbour fill with too small a `capacity` (a supported use of the two-phase
// call) truncates the caller's index array only; lists, forces and a later, larger fill are unaffected.
#define PETAR_ST_FATAL (PETAR_ST_NONFINITE | PETAR_ST_NODE_CAP | PETAR_ST_LIST_CAP | PETAR_ST_STACK)

#define PETAR_MAXLEVEL 21
#define PETAR_NLEVELS 22           // levels 0..21
#define PETAR_CHUNK 1024           // list arena chunk, in 4-byte entries; [0] = next chunk (or -1), [1] unused
#define PETAR_CHUNK_HDR 2
#define PETAR_CHUNK_PAYLOAD (PETAR_CHUNK - PETAR_CHUNK_HDR)   // 1022 entries (even: EP ranges are pairs)
// super-group levels (see SuperRec): level l holds the tree cells with <= PETAR_SUP_LIMIT(l) members
#define PETAR_NSUP 2
#define PETAR_SUP_T0 4096
#define PETAR_SUP_T1 512
#define PETAR_SUP_LIMIT(l) ((l) == 0 ? PETAR_SUP_T0 : PETAR_SUP_T1)
#define PETAR_UNIT_CLASSES 4       // phase-A force units: class 0 = 80..128 particles (tensor-core kernel), then 64, 32 and < 32

// ---- device-resident header (one per tree, lives at the start of the workspace) -----------------
struct DevHeader {
    // encoded bounding box (ordered-uint encoding of doubles) : min x,y,z ; max x,y,z
    unsigned long long bbox[6];
    double c[3];        // root cube centre (O1)
    double h;           // half edge, power of two
    double o[3];        // origin c - h
    double inv_s;       // 2^21 / (2h)
    int n_nodes;
    int n_groups;
    int status;         // PETAR_ST_* bits
    int arena_top;      // next free chunk index
    int level_off[PETAR_NLEVELS + 2];   // node id range of level l: [level_off[l], level_off[l+1])
    int group_ticket;   // dynamic scheduling counters (reset before each consumer kernel)
    int group_ticket2;
    int group_ticket3;
    int n_super[PETAR_NSUP];       // super-groups per level
    int super_ticket[PETAR_NSUP];
    int unit_cnt[PETAR_UNIT_CLASSES];      // force units (phase A) per size class
    int unit_off[PETAR_UNIT_CLASSES + 1];
    int unit_fill[PETAR_UNIT_CLASSES];
    int unit_ticket;
    int unit_ticket_tc;            // k_force_units_tc (class-0 units)
    int n_refine;                  // particles queued for the fp64 re-evaluation (k_force_refine)
    int group_ticket4;             // k_force_near
    int rank_done;                 // k_rank_scan: CTAs (one per level) that have finished; the last one writes level_off and resets it
    unsigned long long n_epep, n_epsp, n_epep_near, n_ep_list, n_sp_list, n_epsp_common;
    unsigned long long nb_total;
};

// node integer record: begin, end, first_child, meta = level | nchild<<8 | leaf<<16 | firstflag<<17
struct __align__(16) NodeInt { int begin, end, first_child, meta; };
// MAC record (fp64, exact decisions): lo[3], hi[3], com[3], rmax  -> 10 doubles = 80 B
struct __align__(16) NodeMac { double lo[3]; double hi[3]; double com[3]; double rmax; };
// fp32 walk record (64 B): conservative pre-test of the MAC; the fp64 NodeMac decides ambiguous cases.
//  a = (lox, loy, loz, hix) ; b = (hiy, hiz, comx, comy) ; c = (comz, rmax, eps, 0) ; d = (begin, end, first_child, meta)
//  coordinates relative to the root centre; eps = 2^-21 * max |box coordinate| bounds the fp32 error (walk.cu)
struct __align__(16) NodeW { float4 a, b, c; int4 d; };
// moments kept for the bottom-up pass / export
struct __align__(16) NodeMom { double M; double S[3]; double Q[6]; };
// fp32 super-particle record for the force kernel: 12 floats = 48 B
//  q0 = (xh, yh, zh, M) ; q1 = (xl, yl, zl, Bxx) ; q2 = (Byy, Bxy, Bxz, Byz) ;  Bzz = -(Bxx + Byy)
//  (xh + xl) = com - c_root in float-float; B = -2 A, A = 1.5 Q - 0.5 tr(Q) I  (Eq. 31, traceless)
struct __align__(16) NodeSp { float4 q0, q1, q2; };

struct __align__(16) GroupRec {
    int begin, end;
    int head_sp, head_epn, head_epf;   // first chunk of each list (-1 = empty)
    int n_sp, n_epn, n_epf;            // entries: cells, near ranges, far ranges
    int n_ep_part, n_epn_part;         // particles in all EP ranges / in near ranges
    int head_spp, n_spp;               // cells closer than the group's own size: float-float ("precise") path
    double lo[3], hi[3], rmax;
    int sid[PETAR_NSUP];               // super-group (see SuperRec) of each level this group lies in
};

// super-group of level l: tree cell with <= PETAR_SUP_LIMIT(l) members (parent has more).  Its walk decides,
// once for all the i-groups inside it, the cells that every one of them accepts ("common" lists) and
// leaves the rest ("deferred" cells) to the next level's walks (level l+1 super-groups, finally the
// i-groups), which start from them instead of from the root.  Records of level l live at
// srec[l * group_cap + id], the map sorted position -> id at smap[l * N + position].
struct __align__(16) SuperRec {
    int node, begin, end;
    int head_sp, n_sp;                 // common cells, group-relative path
    int head_spp, n_spp;               // common cells, float-float path
    int head_def, n_def;               // deferred cells (node ids)
    int pad[3];
};

// phase-A force unit: <= 128 consecutive particles of one super-group against its common cell lists
struct __align__(16) ForceUnit { int rec; int ibeg; int cnt; int level; };

struct Workspace {
    DevHeader* hdr;
    // sort buffers
    unsigned long long *key, *key_alt;
    unsigned int *idx, *idx_alt;
    unsigned int *sort_hist;       // [8][256] global digit totals, then per-pass block counts
    unsigned int *sort_blk;        // [256][nblk]
    double2* rec;                  // [N][4] packed inputs in the caller's order: (x, y), (z, m), (r_out, r_search), -
    // sorted particle data
    double *xs, *ys, *zs, *ms, *routs, *rss;
    double *vxs, *vys, *vzs;       // sorted velocities (petar_neighbor_list_orbit only)
    float4 *pa, *pb;               // (xh,yh,zh,m) , (xl,yl,zl,1/r_out)
    signed char *D;                // [N+1] shared leading octal digits of keys i-1, i
    signed char *depth;            // [N] leaf level of particle i
    signed char *glevel;           // [N] group level
    int *gflag;                    // [N] group-start flags -> scanned
    int *tile_cnt;                 // [22][ntile]
    int *scan_tmp;                 // scan partials
    // nodes
    NodeInt* nint; NodeMac* nmac; NodeMom* nmom; NodeSp* nsp; NodeW* nw;
    int node_cap;
    // groups
    GroupRec* grp; int group_cap;
    SuperRec* srec;                // [PETAR_NSUP][group_cap] super-groups
    int* smap;                     // [PETAR_NSUP][N] sorted position -> super-group id
    struct ForceUnit* units; int unit_cap;   // phase-A force units (force.cu)
    double* part;                  // [PETAR_NSUP + 1][N][4] partial sums (sorted order) ax, ay, az, pot: phase A per super-group level, then the changeover pairs
    double* part_s;                // [PETAR_NSUP + 1][N] cancellation scale (Acc64::s) of the same
    int* refine_q;                 // [N][2] (group, sorted position) of the particles to re-evaluate in fp64
    // list arena
    int* arena; int arena_chunks;
    // neighbour temporaries
    int* nb_cnt;                   // [N] counts in caller's order
    int* nb_queue;                 // [group_cap + 1] groups with a long near list (k_neighbors_big)
    int* exp_scratch;              // [10 (N+1) + 8] list-export scratch (tests)
};

struct petar_tree {
    uint32_t magic;
    int64_t N;
    petar_params p;
    Workspace w;
    const double *x, *y, *z, *m, *r_out, *r_search;
    bool built, walked;
    bool nb_counted;               // w.nb_cnt / w.nb_queue hold the count pass of petar_neighbor_list for this tree (the fill call reuses it)
    cudaEvent_t* ev;               // [2*PETAR_N_STAGES] stage begin/end events (profiling only; created once per handle)
    int stage_rec[PETAR_N_STAGES];
    int sm_count;
    int h_nodes, h_groups;         // host copies of the header counters (filled by petar_debug_export)
    cudaStream_t side;             // second stream: the per-group walk runs beside force phase A (created once per handle)
    cudaEvent_t ev_fork, ev_join, ev_tab;
    void* workspace; size_t workspace_bytes;
};

#define PETAR_MAGIC 0x50335431u

// launch wrappers (each returns cudaError_t of the launch)
cudaError_t launch_keys_sort_gather(petar_tree* t, cudaStream_t s);
cudaError_t launch_tree(petar_tree* t, cudaStream_t s);
cudaError_t launch_walk(petar_tree* t, cudaStream_t s);
cudaError_t launch_walk_supers(petar_tree* t, cudaStream_t s);
cudaError_t launch_walk_groups(petar_tree* t, cudaStream_t s, int ctas_per_sm);
cudaError_t launch_force(petar_tree* t, double* ax, double* ay, double* az, double* pot, cudaStream_t s);
cudaError_t launch_force_units(petar_tree* t, cudaStream_t s);
cudaError_t launch_force_units_table(petar_tree* t, cudaStream_t s);
cudaError_t launch_force_units_tc(petar_tree* t, cudaStream_t s);
cudaError_t launch_force_units_small(petar_tree* t, cudaStream_t s);
cudaError_t launch_force_near(petar_tree* t, cudaStream_t s);
cudaError_t launch_force_groups(petar_tree* t, double* ax, double* ay, double* az, double* pot, cudaStream_t s);
// vx != nullptr: the orbit-dependent two-stage criterion (rule O10) with velocities in the caller's order
cudaError_t launch_neighbors(petar_tree* t, int64_t* offsets, int32_t* indices, int64_t capacity,
                             int32_t* status_dev, cudaStream_t s, const double* vx = nullptr, const double* vy = nullptr,
                             const double* vz = nullptr, double Cv = 0.0);
// stable LSD radix sort of (key, idx) pairs, 8 bits per pass, npass even: the result is back in (key, idx)
cudaError_t launch_radix_sort(unsigned long long* key, unsigned long long* key_alt, unsigned* idx, unsigned* idx_alt,
                              unsigned* hist /* [npass][256] */, unsigned* blk /* [256][nblk] */, long long n, int npass, cudaStream_t s);
int radix_sort_blocks(long long n);
cudaError_t launch_search_radii(const double* vx, const double* vy, const double* vz, const double* r_out, double Cr, double dt,
                                long long n, double* out, cudaStream_t s);
cudaError_t launch_clusters(const long long* offsets, const int* indices, long long n, int* label, long long* n_clusters_dev,
                            long long* cluster_offsets, int* members, void* workspace, cudaStream_t s);
size_t clusters_workspace_bytes(long long n);
cudaError_t launch_export_lists(petar_tree* t, int what, void* dst, size_t dst_bytes, cudaStream_t s);
// device-wide exclusive scan: out[i] = sum_{j<i} in[j], out has n+1 entries (out[n] = total)
cudaError_t launch_scan_i32(const int* in, int* out, int n, int* tmp, cudaStream_t s);
cudaError_t launch_scan_i32_to_i64(const int* in, long long* out, long long n, long long* tmp, cudaStream_t s);

void petar_count_launch(int n);
// PETAR_DEBUG_SYNC=1 in the environment: synchronise after every kernel and report the first failing one
void petar_debug_check(cudaStream_t s, const char* name);
#define KCHECK(s, name) petar_debug_check(s, name)
void stage_begin(petar_tree* t, int stage, cudaStream_t s);
void stage_end(petar_tree* t, int stage, cudaStream_t s);

static inline int cdiv(long long a, long long b) { return (int)((a + b - 1) / b); }

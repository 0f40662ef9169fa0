/*
 * petar.h -- C ABI of the B200-native long-range P3T force path of PeTar (arxiv 2006.16560).
 *
 * What the library computes (citations are PAPER.md:<line>):
 *   For N particles with masses m_i, positions and individual changeover radii r_out,i
 *   (Eq. 12, :226-231), an opening angle theta (:207) and a multipole order (:645):
 *     - the LONG-range acceleration and specific potential of H_L (Eq. 11, :184-187), i.e.
 *       Barnes-Hut tree gravity in which every particle-particle pair is weighted by the paper's
 *       changeover functions, force weight 1-K(x) (Eq. 17, :265) and potential weight 1-W(x)
 *       (Eq. 15, :247), x and Lambda from the pairwise maxima of the radii (Eq. 16, :252-261);
 *     - the neighbour list { j != i : r_ij < max(r_search,i, r_search,j) } that hands particles
 *       to the short-range integrators (:209, :347; r_search = r_out on this path, the
 *       velocity-dependent radius of Eq. 24, :341, can be passed through r_search).
 *
 * Conventions
 *   - Every array pointer is a DEVICE pointer (CUDA global memory of the current device) unless the
 *     parameter comment says HOST.  All particle arrays are SoA, length N, fp64, caller's order.
 *   - The caller owns every input, every output and the workspace; the library never allocates
 *     device memory.  Inputs are read-only and must stay alive (and unmodified) until the stream
 *     has passed the last call that uses the tree.  The tree handle is a small host object that
 *     points into the workspace; it dies with petar_tree_destroy or with the workspace.
 *   - cuda_stream is a cudaStream_t passed as void* (NULL = legacy default stream).  All work is
 *     enqueued on it; calls return without synchronising unless a HOST output is requested.  No call on
 *     the path allocates or frees pinned memory; petar_tree_build creates the small host handle (and, with
 *     profiling on, its CUDA events) once, petar_tree_rebuild reuses it.
 *   - Return value: 0 = PETAR_OK, negative = error (below).  No exceptions, no exit(), no stdout.
 *     Data-dependent failures found on the device (non-finite input, node/list/neighbour capacity
 *     exceeded) are recorded in a device status word, see petar_tree_status.
 */
#ifndef PETAR_H_
#define PETAR_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PETAR_OK 0
#define PETAR_EINVAL (-1)     /* bad N / params / NULL pointer                                   */
#define PETAR_EWORKSPACE (-2) /* workspace too small or misaligned (needs 256-byte alignment)     */
#define PETAR_ECUDA (-3)      /* CUDA launch/runtime error; petar_strerror gives the CUDA text    */
#define PETAR_ENOTBUILT (-4)  /* handle is NULL, destroyed, or no tree has been built into it     */
#define PETAR_ESTATUS (-5)    /* device status word is non-zero (returned only by calls that sync) */
#define PETAR_ECAPACITY (-6)  /* N is larger than the fixed size of the library's built-in scratch array
                                 (petar_short_range_force_noalloc: PETAR_SHORT_RANGE_NOALLOC_MAX_N)    */

/* bits of the device status word */
#define PETAR_ST_NONFINITE 1     /* a position, mass or radius is NaN/Inf, or a radius is <= 0     */
#define PETAR_ST_NODE_CAP 2      /* more tree nodes than the workspace was sized for               */
#define PETAR_ST_LIST_CAP 4      /* interaction-list arena exhausted (lists truncated)             */
#define PETAR_ST_STACK 8         /* walk frontier overflow (never expected)                        */
#define PETAR_ST_NB_CAP 16       /* neighbour indices did not fit `capacity`                       */

typedef struct petar_tree petar_tree; /* opaque */

typedef struct {
    double G;               /* gravitational constant; 1.0 in Henon units (:580, :625)              */
    double theta;           /* opening angle (:207); 0 => every leaf opened => direct summation     */
    double r_in_over_r_out; /* r_in/r_out, in (0,1); the paper fixes 0.1 (:650)                     */
    int32_t multipole;      /* 1 = monopole, 2 = quadrupole super-particles (:645)                  */
    int32_t n_leaf_limit;   /* leaf capacity of the octree, 1..64 (8)                               */
    int32_t n_group_limit;  /* i-group capacity, n_leaf_limit..64 (64)                              */
    int32_t flags;          /* reserved, must be 0                                                  */
    double list_entries_per_particle; /* sizing of the interaction-list arena in 4-byte entries per
                               particle; <= 0 selects the default (see petar_workspace_bytes)       */
    double nodes_per_particle; /* sizing of the node table: capacity = nodes_per_particle * N + 4096; <= 0
                               selects the default (1 for n_leaf_limit >= 4, else 3).  The octree keeps
                               single-child chains (rule O5), so deep tight binaries with small leaves can
                               need more: PETAR_ST_NODE_CAP reports it, this field raises the capacity     */
} petar_params;

/* Interaction counters (HOST struct).  Self pairs are counted in n_epep, as in rule O7.            */
typedef struct {
    int64_t n_groups, n_nodes;
    int64_t n_epep;         /* sum over groups n_i * n_ep   (particle-particle interactions)        */
    int64_t n_epsp;         /* sum over groups n_i * n_sp   (particle-cell interactions)            */
    int64_t n_epep_near;    /* part of n_epep that went through the changeover polynomials          */
    int64_t n_ep_list;      /* sum over groups of EP particle ranges as listed: near leaves one range each,
                               runs of contiguous far leaves joined into one range (<= the number of leaves) */
    int64_t n_sp_list;      /* sum over groups of accepted cells                                    */
    int64_t list_entries_used; /* 4-byte arena entries used                                         */
    int64_t n_epsp_common;  /* part of n_epsp evaluated super-group-wide (cells every i-group of a
                               super-group accepts; force phase A)             */
    int64_t n_refined;      /* particles whose force nearly cancels (|a| < 2e-3 of the summed magnitudes) and
                               was therefore re-evaluated in fp64                */
} petar_counts;

/* HOST-only query: bytes of device workspace petar_tree_build needs for N particles.
 * Returns 0 if N < 0 or the parameters are invalid.  Sized for: sorted copies of the inputs, keys,
 * the node table (capacity nodes_per_particle * N + 4096 nodes), group table and
 * the list arena (default 1024 entries per particle, at least 16 Mi entries).                        */
size_t petar_workspace_bytes(int64_t N, const petar_params* p /* HOST */);

/* Steps S0-S6 of the path: bounding cube, 63-bit Morton keys, stable radix sort, sorted SoA copies,
 * octree (leaf iff count <= n_leaf_limit or level 21), bottom-up monopole/quadrupole moments with
 * tight boxes, i-groups (tree cells with <= n_group_limit members).  The paper delegates this to
 * FDPS (:195, :615); the rules are DESIGN.md's readings O1-O6.
 *   x,y,z,m,r_out : DEVICE fp64[N]; r_out > 0.   r_search: DEVICE fp64[N] or NULL (=> r_out);
 *                   must be >= r_out elementwise if given.
 *   workspace     : DEVICE, 256-byte aligned, >= petar_workspace_bytes(N,p) bytes.
 *   tree_out      : HOST, receives the handle (also for N == 0).
 * Errors: PETAR_EINVAL, PETAR_EWORKSPACE, PETAR_ECUDA.                                              */
int petar_tree_build(const double* x, const double* y, const double* z, const double* m,
                     const double* r_out, const double* r_search, int64_t N,
                     const petar_params* p /* HOST */, void* workspace, size_t workspace_bytes,
                     void* cuda_stream, petar_tree** tree_out /* HOST */);

/* The same steps into an EXISTING handle: same N, parameters and workspace as the petar_tree_build that
 * created it, new (or moved) particle arrays.  Nothing is allocated, created or synchronised; lists and
 * results of the previous tree are invalidated.  This is the call of a time-stepping loop.
 * Errors: PETAR_ENOTBUILT (bad handle), PETAR_EINVAL (NULL array), PETAR_ECUDA.                     */
int petar_tree_rebuild(petar_tree* t, const double* x, const double* y, const double* z, const double* m,
                       const double* r_out, const double* r_search, void* cuda_stream);

/* Steps S7-S8: per-group interaction-list walk (cell forced open when its box comes within
 * max(rmax_group, rmax_cell) of the group's box, else accepted iff edge < theta * distance, rule O7)
 * and the fp32 pairwise force + potential kernel (rule O8) with the changeover weights (Eq. 15-17).
 *   acc_x, acc_y, acc_z, pot : DEVICE fp64[N], caller's particle order; pot is the specific
 *                              long-range potential phi_L,i (negative).  Any may be NULL (skipped).
 *   counts_host_or_null      : HOST; if non-NULL the call synchronises the stream and fills it, and
 *                              returns PETAR_ESTATUS if one of the status bits named below is set.
 * When PETAR_ST_NONFINITE, _NODE_CAP, _LIST_CAP or _STACK is set (the tree or its lists are unusable) the force
 * kernels write NOTHING: the outputs keep their previous contents; check petar_tree_status (or pass counts) before
 * using them.  PETAR_ST_NB_CAP (a neighbour fill whose `capacity` was too small) does not affect this call.
 * Errors: PETAR_ENOTBUILT, PETAR_ECUDA, PETAR_ESTATUS.                                              */
int petar_long_range_force(petar_tree* t, double* acc_x, double* acc_y, double* acc_z, double* pot,
                           petar_counts* counts_host_or_null, void* cuda_stream);

/* Step S9: compacted neighbour list in CSR form, caller's particle indices (rule O9, fp64 test
 * r2 < R_ij^2 with R_ij = max(r_search,i, r_search,j), strict).
 *   offsets    : DEVICE int64[N+1]; always written; offsets[N] = total number of neighbours.
 *   indices    : DEVICE int32[capacity] or NULL.  NULL => only offsets (count + scan) are written;
 *                the caller reads offsets[N], allocates, and calls again (two-phase output).  The per-particle counts of
 *                the first call are kept in the workspace until the next (re)build or _orbit call: the second call only scans and fills.
 *   status_dev : DEVICE int32[1] or NULL; set to 0, or 1 if offsets[N] > capacity (then rows that
 *                do not fit are not written).
 * Row order is deterministic but unspecified (compare rows as sets).
 * Errors: PETAR_ENOTBUILT, PETAR_EINVAL (capacity < 0), PETAR_ECUDA.                                */
int petar_neighbor_list(petar_tree* t, int64_t* offsets, int32_t* indices, int64_t capacity,
                        int32_t* status_dev, void* cuda_stream);

/* ---- the consumers of the neighbour search --------------------------------
 * Eq. 24: r_search_out[i] = r_out[i] + C_r |v_i| dt_L  (C_r = 3 in the paper); the result
 * is what petar_tree_build takes as r_search.  All arrays DEVICE fp64[N]; r_search_out may not alias.
 * Errors: PETAR_EINVAL (N < 0, C_r < 0, dt_L < 0, NULL), PETAR_ECUDA.                                */
int petar_search_radii(const double* vx, const double* vy, const double* vz, const double* r_out,
                       double C_r, double dt_L, int64_t N, double* r_search_out, void* cuda_stream);

/* Orbit-dependent two-stage neighbour criterion (DESIGN.md rule O10, reading P20) on a
 * tree built with r_search = the Eq. 24 radii:  j is a neighbour of i iff j != i,
 *   (i)  r_ij < max(r_search,i, r_search,j)                       (the candidates of rule O9) and
 *   (ii) r_ij < max(r_out,i, r_out,j)  or  r_p,ij < C_V min(r_search,i, r_search,j),
 * r_p,ij = pericentre separation of the pair's two-body Kepler orbit, mu = G (m_i + m_j), fp64.
 *   vx, vy, vz : DEVICE fp64[N], caller's particle order.   C_V >= 0 (1.5 in the paper).
 * Output, two-phase protocol, ownership and errors as petar_neighbor_list.                          */
int petar_neighbor_list_orbit(petar_tree* t, const double* vx, const double* vy, const double* vz, double C_V,
                              int64_t* offsets, int32_t* indices, int64_t capacity, int32_t* status_dev,
                              void* cuda_stream);

/* Clustering: connected components of a symmetric neighbour list in CSR form.
 *   offsets int64[N+1], indices int32[offsets[N]] : DEVICE, as written by petar_neighbor_list(_orbit).
 *   label            : DEVICE int32[N]; label[i] = smallest particle index of i's cluster.
 *   n_clusters_dev   : DEVICE int64[1] or NULL.
 *   cluster_offsets  : DEVICE int64[N+1] or NULL.  If given, the clusters are numbered by ascending label,
 *                      cluster c holds members[cluster_offsets[c] .. cluster_offsets[c+1]) in ascending
 *                      particle index, cluster_offsets[n_clusters] = N (entries beyond are untouched).
 *   members          : DEVICE int32[N] or NULL (needs cluster_offsets).
 *   workspace        : DEVICE, 256-byte aligned, >= petar_clusters_workspace_bytes(N); only read when
 *                      cluster_offsets is given.
 * No host synchronisation.  Errors: PETAR_EINVAL, PETAR_EWORKSPACE, PETAR_ECUDA.                     */
size_t petar_clusters_workspace_bytes(int64_t N);
int petar_clusters(const int64_t* offsets, const int32_t* indices, int64_t N, int32_t* label,
                   int64_t* n_clusters_dev, int64_t* cluster_offsets, int32_t* members,
                   void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Short-range part H_S of Eq. 11 over neighbour rows: for every i
 *   a_S,i = -G sum_j m_j K(x) d/r^3,   j_S,i = d a_S,i / dt,   phi_S,i = -G sum_j m_j W(x)/r,   j in row i,
 * d = x_i - x_j, K, W of Eq. 17 / Eq. 15 with R = max(r_out,i, r_out,j), r_in = r_in_over_r_out * R and
 * K' = -280 Lambda (x+q) x^3 (1-x)^3 (from Eq. 18) in the jerk.  Entries at r >= R or r = 0 contribute nothing.
 *   x..r_out      : DEVICE fp64[N], caller's order (the order the neighbour list refers to).
 *   offsets, indices : DEVICE CSR neighbour list (petar_neighbor_list / _orbit).
 *   acc_*, jerk_*, pot : DEVICE fp64[N]; any may be NULL (skipped).  fp64 throughout; rows are summed in
 *                    list order (rows longer than 32 entries by one warp, in a fixed order).
 *   workspace     : DEVICE, 256-byte aligned, >= petar_short_range_workspace_bytes(N).
 * No host synchronisation.  Errors: PETAR_EINVAL, PETAR_EWORKSPACE, PETAR_ECUDA.                    */
size_t petar_short_range_workspace_bytes(int64_t N);
int petar_short_range_force(const double* x, const double* y, const double* z,
                            const double* vx, const double* vy, const double* vz,
                            const double* m, const double* r_out,
                            const int64_t* offsets, const int32_t* indices, int64_t N,
                            double G, double r_in_over_r_out,
                            double* acc_x, double* acc_y, double* acc_z,
                            double* jerk_x, double* jerk_y, double* jerk_z, double* pot,
                            void* workspace, size_t workspace_bytes, void* cuda_stream);

/* The same computation, same arguments and same results as petar_short_range_force, for callers that cannot
 * give it a workspace because they cannot allocate device memory at all: code that runs as a plug-in of a host
 * application and is only ever handed pointers; code inside a memory pool whose budget is fixed and spent; a
 * latency-bound integrator loop that must not hit the device-wide synchronisation of cudaMalloc/cudaFree.  Such a
 * caller passes its inputs and outputs and nothing else.
 *
 * Where the scratch lives.  The packed particle records and the queue of long rows (68 bytes per particle) go to a
 * fixed array that is part of the library itself, sized for PETAR_SHORT_RANGE_NOALLOC_MAX_N particles (about
 * 4.3 MB).  The cost of that convenience: every GPU that loads this library holds the array until the process
 * exits, called or not.  N above the maximum is refused with PETAR_ECAPACITY before anything is enqueued; use
 * petar_short_range_force with your own workspace for larger sets.
 *
 * The call itself never calls cudaMalloc, cudaFree or any other allocating routine (one 4-byte cudaMemsetAsync,
 * three kernel launches).  The FIRST call on each device also looks up the array's device address (the device of the
 * stream must be the current device, as for every call of this library); make that first call outside any stream
 * capture, e.g. once at start-up with a tiny N.  Later calls on that device only launch.
 *
 * One array for everybody.  All calls in the process on one device share the array and it keeps whatever the last
 * call left in it; the call clears the one counter that has to start at zero.  Two calls that can be in flight on
 * the GPU at the same time (different streams, or different host threads on different streams) write over each
 * other's scratch and give wrong results: put them on one stream, or order them with events.
 * Errors: PETAR_EINVAL, PETAR_ECAPACITY, PETAR_ECUDA.                                                 */
#define PETAR_SHORT_RANGE_NOALLOC_MAX_N 65536
int petar_short_range_force_noalloc(const double* x, const double* y, const double* z,
                                    const double* vx, const double* vy, const double* vz,
                                    const double* m, const double* r_out,
                                    const int64_t* offsets, const int32_t* indices, int64_t N,
                                    double G, double r_in_over_r_out,
                                    double* acc_x, double* acc_y, double* acc_z,
                                    double* jerk_x, double* jerk_y, double* jerk_z, double* pot,
                                    void* cuda_stream);

/* ---- P3T-kick and the artificial particles (section 6.4) -----------
 * P3T-kick: v += a dt, in place.  All DEVICE fp64[N].                           */
int petar_kick(double* vx, double* vy, double* vz, const double* ax, const double* ay, const double* az,
               double dt, int64_t N, void* cuda_stream);

/* Artificial particles of n_bin binaries.  pairs: DEVICE int32[n_bin][2], the particle indices
 * of the two members.  For binary b the outputs hold PETAR_ART_COUNT(order) entries starting at
 * b * PETAR_ART_COUNT(order):
 *   [0, n_tt)       tidal-tensor measure points, mass 0: the corners of a regular tetrahedron (order 2, n_tt = 4)
 *                   or of the paper's "cube" (order 3, n_tt = 8) around the centre of mass, coordinates of
 *                   Table 1 part (3) times d_c = tt_scale * a (reading P24);
 *   [n_tt]          the centre-of-mass point, mass 0 (it measures A(r_cm), Eq. 27);
 *   [n_tt+1, +3)    the pseudoparticles of Eq. 38, mass (m1+m2)/3 each, in the orbital frame of Eq. 32 (x to
 *                   the pericentre, z along the angular momentum) around the centre of mass.
 *   elem : DEVICE fp64[n_bin][8] or NULL: a, e, d_c, cm[3], bound (1/0), m1+m2.
 * An unbound or radial pair gets bound = 0, d_c = 0 and every entry at the centre of mass (the three masses
 * still carry the monopole).  The caller appends the entries to the particle set for the tree build and gives the
 * members zero mass there.  Errors: PETAR_EINVAL (order not 2 | 3, tt_scale <= 0, G <= 0, NULL), PETAR_ECUDA. */
#define PETAR_ART_COUNT(order) ((order) == 2 ? 8 : 12)
#define PETAR_TT_COEFFS(order) ((order) == 2 ? 6 : 16)
int petar_artificial_particles(const double* x, const double* y, const double* z,
                               const double* vx, const double* vy, const double* vz, const double* m,
                               const int32_t* pairs, int64_t n_bin, double G, int32_t order, double tt_scale,
                               double* art_x, double* art_y, double* art_z, double* art_m,
                               double* elem, void* cuda_stream);

/* Orbit-sampling particles (Eq. 29): for binary b, out_*[b * 2 n_split ...] hold n_split samples
 * of component 1 and then n_split of component 2, at eccentric anomalies E_k = k * 2 pi / n_split (reading P27),
 * positions by Eq. 32-33 in the orbital frame around the centre of mass, masses m_i dM_k / (2 pi),
 * dM_k = dE - 2 e cos(E_k) sin(dE / 2).  An unbound pair puts every sample at the centre of mass with mass
 * m_i / n_split.  1 <= n_split <= 1024 (8 in the paper: "16 particles").  Errors as above.               */
int petar_orbit_sampling(const double* x, const double* y, const double* z,
                         const double* vx, const double* vy, const double* vz, const double* m,
                         const int32_t* pairs, int64_t n_bin, double G, int32_t n_split,
                         double* out_x, double* out_y, double* out_z, double* out_m, void* cuda_stream);

/* Tidal-tensor coefficients (Eq. 25-26) from the long-range accelerations measured at the artificial particles
 * (acc_*: DEVICE fp64, same layout as art_*): T[b] = M^-1 (A(r_k) - A(r_cm)), M^-1 the generalized inverse of
 * Eq. 28 = the formulas of Table 1 part (1).  T: DEVICE fp64[n_bin][PETAR_TT_COEFFS(order)], order
 * xx xy xz yy yz zz [xxx xxy xxz xyy xyz xzz yyy yyz yzz zzz]; convention of Table 1 part (2):
 * A_i(r) = A_i(r_cm) + A_ij r'_j + A_ijk r'_j r'_k.  Binaries with d_c = 0 get zeros.                 */
int petar_tidal_tensor_fit(const double* acc_x, const double* acc_y, const double* acc_z, const double* elem,
                           int64_t n_bin, int32_t order, double* T, void* cuda_stream);

/* Synchronises the stream and returns the device status word (PETAR_ST_* bits) in *status_host.    */
int petar_tree_status(petar_tree* t, int32_t* status_host /* HOST */, void* cuda_stream);

/* Invalidates and frees the HOST handle (the workspace stays the caller's).  NULL is allowed.      */
int petar_tree_destroy(petar_tree* t);

/* Static text for an error code; for PETAR_ECUDA the text of the last CUDA error seen.             */
const char* petar_strerror(int code);

/* ---- test hooks (not part of the timed path) ---------------------------------------------------
 * petar_debug_export copies an intermediate to `dst` (DEVICE, dst_bytes) and synchronises.
 * Layouts (n = N, nn = n_nodes, ng = n_groups; nodes in (level, begin) order, which is the
 * library's own node numbering):
 *   PETAR_DBG_HEADER   int64[8]  : n_nodes, n_groups, status, arena entries used, 0...
 *   PETAR_DBG_ROOT     double[4] : root cube centre c[3], half edge h
 *   PETAR_DBG_KEYS     uint64[n] : sorted Morton keys
 *   PETAR_DBG_PERM     int32[n]  : sorted position -> caller's index
 *   PETAR_DBG_NODE_INT int32[nn*4]: begin, end, first_child, level | nchild<<8 | leaf<<16
 *   PETAR_DBG_NODE_DBL double[nn*17]: M, com[3], lo[3], hi[3], rmax, Q[6] (xx yy zz xy xz yz about com)
 *   PETAR_DBG_GROUP_INT int32[ng*2]: begin, end
 *   PETAR_DBG_GROUP_DBL double[ng*7]: lo[3], hi[3], rmax
 *   PETAR_DBG_GROUP_CNT int32[ng*4]: n_sp, n_ep ranges (near), n_ep ranges (far), n_ep particles
 *   PETAR_DBG_GROUP_SUPER int32[ng*8]: for each of the two super-group levels: super-group id, its
 *                        particle count, cells its walk accepted for all of its groups ("common"
 *                        cells, part of n_sp above), cells it deferred
 *   PETAR_DBG_LIST_OFFS int64[ng*3+1]: start of each group's SP / near-EP / far-EP block in the
 *                        flattened list below, in 4-byte entries; last = total
 *   PETAR_DBG_LISTS    int32[total]: SP node ids; EP ranges as (begin, end) pairs
 * The LIST_* exports require a prior petar_long_range_force or petar_neighbor_list on the tree.     */
#define PETAR_DBG_HEADER 0
#define PETAR_DBG_ROOT 1
#define PETAR_DBG_KEYS 2
#define PETAR_DBG_PERM 3
#define PETAR_DBG_NODE_INT 4
#define PETAR_DBG_NODE_DBL 5
#define PETAR_DBG_GROUP_INT 6
#define PETAR_DBG_GROUP_DBL 7
#define PETAR_DBG_GROUP_CNT 8
#define PETAR_DBG_LIST_OFFS 9
#define PETAR_DBG_LISTS 10
#define PETAR_DBG_GROUP_SUPER 11
int petar_debug_export(petar_tree* t, int what, void* dst, size_t dst_bytes, void* cuda_stream);

/* Per-stage device times of the last build / force / neighbour call on this tree, in ms, measured
 * with CUDA events when profiling was switched on with petar_set_profiling(1) (HOST; default off;
 * it must be set before petar_tree_build; events are recorded asynchronously and petar_stage_times synchronises on them).  stage_ms: HOST float[PETAR_N_STAGES].             */
#define PETAR_STAGE_BBOX_KEYS 0
#define PETAR_STAGE_SORT 1
#define PETAR_STAGE_GATHER 2
#define PETAR_STAGE_TREE 3
#define PETAR_STAGE_MOMENTS 4
#define PETAR_STAGE_GROUPS 5
#define PETAR_STAGE_WALK 6
#define PETAR_STAGE_FORCE 7
#define PETAR_STAGE_NEIGHBOR 8
#define PETAR_STAGE_FORCE_UNITS 9   /* force phase A: a two-stream STAGE (unit table + k_force_units_tc on the caller's stream;
                                       on a first force call also k_walk, k_force_units, k_force_near on the side stream).
                                       PETAR_STAGE_FORCE is phase B: the event pair spans the single k_force launch          */
#define PETAR_STAGE_WALK_SUPER 10   /* super-group walks; PETAR_STAGE_WALK is the per-group walk (k_walk)   */
#define PETAR_STAGE_FORCE_REFINE 11 /* k_force_refine: fp64 re-evaluation of the n_refined near-cancelling particles  */
#define PETAR_N_STAGES 12
int petar_set_profiling(int on);
int petar_stage_times(petar_tree* t, float* stage_ms /* HOST */);
/* Number of kernel launches the library has enqueued since process start (HOST counter).           */
int64_t petar_launch_count(void);

/* Measurement hook (not part of the path): enqueues an FFMA-only kernel (16 independent chains per
 * thread, 8 CTAs x 256 threads per SM) and returns the flops it executes in *flops_out_host (HOST);
 * the caller times it with CUDA events to obtain this GPU's CUDA-core FP32 peak.
 * scratch_dev: DEVICE float[1].                                                                      */
int petar_probe_fp32(int64_t iters, double* flops_out_host, float* scratch_dev, void* cuda_stream);
#ifdef __cplusplus
}
#endif
#endif /* PETAR_H_ */

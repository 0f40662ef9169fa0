// walk.cu -- step S7 (interaction-list walk, rule O7: two super-group levels, then the i-groups), step S9
// (neighbour-list writer, rules O9 / O10) and the list export used by the tests.  Compiled with -fmad=false: the MAC and the
// neighbour test are fp64 with exactly the operation order of DESIGN.md O7 / O9 (fma where written).
#include "internal.cuh"

#define WALK_WARPS 8
#define WALK_STACK 1504          // frontier entries per warp (shared memory) of the super-group walks
#define GWALK_STACK 640          // ... of the per-group walk (it starts from short deferred lists; 20 KB per CTA let two of its CTAs share an SM with two CTAs of k_force_units_tc)

// warp-uniform cursor of one chunked list
struct ListCursor {
    int head;      // first chunk or -1
    int chunk;     // current chunk or -1
    int pos;       // payload entries used in the current chunk
    int dead;      // arena exhausted
};

// Appends `per` entries (1 or 2) for every lane with `take` set.  v0/v1 are the lane's entries.
__device__ __forceinline__ void list_append(ListCursor& c, bool take, int per, int v0, int v1, int* __restrict__ arena,
                                            int arena_chunks, DevHeader* __restrict__ h, int lane) {
    const unsigned mask = __ballot_sync(0xffffffffu, take);
    if (mask == 0u || c.dead) return;
    const int n = __popc(mask);
    int off = __popc(mask & ((1u << lane) - 1u)) * per;        // my first slot relative to c.pos
    int space = (c.chunk >= 0) ? (PETAR_CHUNK_PAYLOAD - c.pos) : 0;
    // part 1: what fits into the current chunk
    if (take && off < space) {
        int* p = arena + (size_t)c.chunk * PETAR_CHUNK + PETAR_CHUNK_HDR + c.pos + off;
        p[0] = v0;
        if (per == 2) p[1] = v1;
    }
    if (n * per <= space) { c.pos += n * per; return; }
    // part 2: new chunk for the rest
    int nc = 0;
    if (lane == 0) {
        nc = atomicAdd(&h->arena_top, 1);
        if (nc >= arena_chunks) { atomicOr(&h->status, PETAR_ST_LIST_CAP); nc = -1; }
        else {
            arena[(size_t)nc * PETAR_CHUNK] = -1;
            if (c.chunk >= 0) arena[(size_t)c.chunk * PETAR_CHUNK] = nc;
        }
    }
    nc = __shfl_sync(0xffffffffu, nc, 0);
    if (nc < 0) { c.dead = 1; return; }
    if (c.chunk < 0) c.head = nc;
    c.chunk = nc;
    if (take && off >= space) {
        int* p = arena + (size_t)nc * PETAR_CHUNK + PETAR_CHUNK_HDR + (off - space);
        p[0] = v0;
        if (per == 2) p[1] = v1;
    }
    c.pos = n * per - space;
}

// ------------------------------------------------------------------------------------------------
// Super-groups.  A node is a level-l super-group iff (count <= T_l or it is a leaf) and its parent
// holds more than T_l particles (or it is the root).  T_l >= n_group_limit, so every i-group lies inside
// exactly one super-group of every level, and a level-(l+1) super-group inside exactly one of level l.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_super_collect(DevHeader* __restrict__ h, const NodeW* __restrict__ nw,
                                                       const unsigned long long* __restrict__ key, long long n,
                                                       SuperRec* __restrict__ srec, int node_cap, int lvl, int limit) {
    const int nn = h->n_nodes;
    if (nn > node_cap) return;
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= nn) return;
    const int4 d = nw[id].d;
    const int level = d.w & 255;
    const bool leaf = (d.w >> 16) & 1;
    if (!(d.y - d.x <= limit || leaf)) return;
    if (level > 0) {
        // parent's particle count: the range of keys that share the level-1 prefix of this cell
        const int shift = 3 * (PETAR_MAXLEVEL - (level - 1));
        const unsigned long long pref = (level - 1 > 0) ? (key[d.x] >> shift) : 0ull;
        long long lo = 0, hi = d.x;                 // first index whose prefix equals pref
        while (lo < hi) { long long mid = (lo + hi) >> 1; if (((level - 1 > 0) ? (key[mid] >> shift) : 0ull) < pref) lo = mid + 1; else hi = mid; }
        const long long pb = lo;
        lo = d.y; hi = n;                           // first index whose prefix exceeds pref
        while (lo < hi) { long long mid = (lo + hi) >> 1; if (((level - 1 > 0) ? (key[mid] >> shift) : 0ull) <= pref) lo = mid + 1; else hi = mid; }
        if (lo - pb <= limit) return;               // an ancestor is the super-group
    }
    const int sid = atomicAdd(&h->n_super[lvl], 1);
    SuperRec r;
    r.node = id; r.begin = d.x; r.end = d.y;
    r.head_sp = r.head_spp = r.head_def = -1; r.n_sp = r.n_spp = r.n_def = 0;
    r.pad[0] = r.pad[1] = r.pad[2] = 0;
    srec[sid] = r;
}

__global__ void __launch_bounds__(256) k_super_map(const DevHeader* __restrict__ h, const SuperRec* __restrict__ srec, int* __restrict__ smap, int lvl) {
    const int lane = threadIdx.x & 31;
    const int ns = h->n_super[lvl];
    for (int s = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; s < ns; s += (gridDim.x * blockDim.x) >> 5)
        for (int p = srec[s].begin + lane; p < srec[s].end; p += 32) smap[p] = s;
}

// fp64 MAC of rule O7 (exactly this operation order); returns act: 0 SP, 1 EP near, 2 EP far, 3 open
__device__ __noinline__ int mac_exact(const NodeMac* __restrict__ cp, const int level, const bool leaf,
                                      const GroupRec* __restrict__ gr, const double theta, const double twoh) {
    const NodeMac c = *cp;
    const double glo0 = gr->lo[0], glo1 = gr->lo[1], glo2 = gr->lo[2];
    const double ghi0 = gr->hi[0], ghi1 = gr->hi[1], ghi2 = gr->hi[2];
    const double grmax = gr->rmax;
    const double theta2 = theta * theta;
    double gx = fmax(0.0, fmax(c.lo[0] - ghi0, glo0 - c.hi[0]));
    double gy = fmax(0.0, fmax(c.lo[1] - ghi1, glo1 - c.hi[1]));
    double gz = fmax(0.0, fmax(c.lo[2] - ghi2, glo2 - c.hi[2]));
    double d2box = fma(gz, gz, fma(gy, gy, gx * gx));
    double R = fmax(grmax, c.rmax);
    bool nearb = d2box < R * R;
    double px = fmax(0.0, fmax(glo0 - c.com[0], c.com[0] - ghi0));
    double py = fmax(0.0, fmax(glo1 - c.com[1], c.com[1] - ghi1));
    double pz = fmax(0.0, fmax(glo2 - c.com[2], c.com[2] - ghi2));
    double d2com = fma(pz, pz, fma(py, py, px * px));
    double edge = ldexp(twoh, -level);
    bool farb = (edge * edge) < theta2 * d2com;
    if (!nearb && farb) return 0;
    if (leaf) return nearb ? 1 : 2;
    return 3;
}

// The walk decides every cell in fp32 first, with a rigorous error band, and falls back to the fp64
// test of rule O7 only when the fp32 values cannot decide (so the decisions are exactly O7's).
// fp32 coordinates q32 = fl32(q - c_root) carry |error| <= 2^-24 |q - c_root|.  With A_c, A_g the largest
// |coordinate| of the cell's / group's box, a computed distance differs from the exact one by less than
// 8 * 2^-24 (A_c + A_g) = eps_c + eps_g (component differences: 2(u_c+u_g) each; norm: 2 sqrt(3)(u_c+u_g);
// rounding of the sum of squares: < 2.6 (u_c+u_g)); thresholds get a further relative 2^-22 for their own
// rounding and the fp32 conversion of rmax and of the per-level edge/theta.
#define WALK_RESERVE 160
// Walk of one super-group S (one warp each).  All tests are fp32 with the error band described below
// and only DEFINITE outcomes are used, so the result is sound for every i-group g inside S:
//   accepted for S  (box(S) not within R of the cell, edge < theta * dist(box(S), com))  =>  accepted by every g,
//        because box(g) is inside box(S): both distances can only grow and rmax_g <= rmax_S;
//   edge >= theta * (largest distance from com to a corner of box(S))  =>  not "far" for any g  =>  opened by every g;
//   anything else (and every leaf) is DEFERRED to the per-group walks.
// Hence the cells a group accepts are exactly S's common cells plus what its own walk finds below the
// deferred cells - the same set rule O7 gives when walked from the root.
// A super-group of level l > 0 starts from the cells its level-(l-1) super-group deferred (psrec / psmap);
// level 0 starts from the root.
__global__ void __launch_bounds__(WALK_WARPS * 32) k_walk_super(DevHeader* __restrict__ h, const NodeW* __restrict__ nw,
                                                                SuperRec* __restrict__ srec, const SuperRec* __restrict__ psrec,
                                                                const int* __restrict__ psmap, int* __restrict__ arena, int arena_chunks,
                                                                double theta, int node_cap, int lvl) {
    __shared__ int s_stack[WALK_WARPS][WALK_STACK];
    __shared__ float s_lt[PETAR_NLEVELS];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int* stack = s_stack[w];
    const int ns = h->n_super[lvl];
    if (h->n_nodes > node_cap || h->n_nodes <= 0) return;
    const double twoh = 2.0 * h->h;
    if (threadIdx.x < PETAR_NLEVELS) s_lt[threadIdx.x] = (theta > 0.0) ? (float)(ldexp(twoh, -(int)threadIdx.x) / theta) : INFINITY;
    __syncthreads();
    for (;;) {
        int s = 0;
        if (lane == 0) s = atomicAdd(&h->super_ticket[lvl], 1);
        s = __shfl_sync(0xffffffffu, s, 0);
        if (s >= ns) break;
        const NodeW sb = nw[srec[s].node];           // the super-group's own cell: tight box, rmax, eps
        const float fl0 = sb.a.x, fl1 = sb.a.y, fl2 = sb.a.z, fh0 = sb.a.w, fh1 = sb.b.x, fh2 = sb.b.y;
        const float frm = sb.c.y, geps = sb.c.z;
        const float gedge = fmaxf(fh0 - fl0, fmaxf(fh1 - fl1, fh2 - fl2));
        const float gedge2 = gedge * gedge;
        ListCursor lsp = {-1, -1, 0, 0}, lspp = {-1, -1, 0, 0}, ldef = {-1, -1, 0, 0};
        int n_sp = 0, n_spp = 0, n_def = 0;
        int top = 0, dchunk = -1, dremaining = 0, doff = 0;
        if (psrec) { const SuperRec* pr = &psrec[psmap[srec[s].begin]]; dchunk = pr->head_def; dremaining = pr->n_def; }
        else { top = 1; if (lane == 0) stack[0] = 0; }
        __syncwarp();
        while (top > 0 || dremaining > 0) {
            if (top == 0) {                    // frontier empty: take the next (up to 256) cells the parent deferred
                if (dchunk < 0) break;         // truncated list (arena exhausted, PETAR_ST_LIST_CAP is set)
                const int* cp = arena + (size_t)dchunk * PETAR_CHUNK;
                const int k = min(256, min(dremaining, PETAR_CHUNK_PAYLOAD - doff));
                for (int e = lane; e < k; e += 32) stack[e] = cp[PETAR_CHUNK_HDR + doff + e];
                top = k; dremaining -= k; doff += k;
                if (dremaining > 0 && doff >= PETAR_CHUNK_PAYLOAD) { dchunk = cp[0]; doff = 0; }
                __syncwarp();
            }
            int p = min(32, top);
            if (top + 7 * p > WALK_STACK - WALK_RESERVE) p = max(1, min(p, (WALK_STACK - WALK_RESERVE - top) / 7));
            const int node = (lane < p) ? stack[top - p + lane] : -1;
            top -= p;
            __syncwarp();
            int act = -1;                      // 0 common (plain), 4 common (precise), 3 open, 5 deferred
            int fc = 0, nch = 0;
            if (node >= 0) {
                const NodeW c = nw[node];
                const int meta = c.d.w;
                const int level = meta & 255;
                const bool leaf = (meta >> 16) & 1;
                fc = c.d.z; nch = (meta >> 8) & 15;
                const float gx = fmaxf(0.f, fmaxf(c.a.x - fh0, fl0 - c.a.w));
                const float gy = fmaxf(0.f, fmaxf(c.a.y - fh1, fl1 - c.b.x));
                const float gz = fmaxf(0.f, fmaxf(c.a.z - fh2, fl2 - c.b.y));
                const float d2b = fmaf(gz, gz, fmaf(gy, gy, gx * gx));
                const float px = fmaxf(0.f, fmaxf(fl0 - c.b.z, c.b.z - fh0));
                const float py = fmaxf(0.f, fmaxf(fl1 - c.b.w, c.b.w - fh1));
                const float pz = fmaxf(0.f, fmaxf(fl2 - c.c.x, c.c.x - fh2));
                const float d2c = fmaf(pz, pz, fmaf(py, py, px * px));
                const float mx = fmaxf(fabsf(c.b.z - fl0), fabsf(fh0 - c.b.z));
                const float my = fmaxf(fabsf(c.b.w - fl1), fabsf(fh1 - c.b.w));
                const float mz = fmaxf(fabsf(c.c.x - fl2), fabsf(fh2 - c.c.x));
                const float dmax2 = fmaf(mz, mz, fmaf(my, my, mx * mx));
                const float D = geps + c.c.z;
                const float R = fmaxf(frm, c.c.y);
                const float Dr = fmaf(R, 2.4e-7f, D);
                const float Rp = R + Dr;
                const bool near_no = d2b > Rp * Rp;
                const float L = s_lt[level];
                const float Dl = fmaf(L, 2.4e-7f, D);
                const float Lm = fmaxf(L - Dl, 0.f), Lp = L + Dl;
                const bool far_yes = d2c > Lp * Lp;
                const bool open_all = !leaf && (dmax2 < Lm * Lm);
                if (near_no && far_yes) act = (d2b < gedge2) ? 4 : 0;
                else if (open_all) act = 3;
                else act = 5;
            }
            list_append(lsp, act == 0, 1, node, 0, arena, arena_chunks, h, lane);
            list_append(lspp, act == 4, 1, node, 0, arena, arena_chunks, h, lane);
            list_append(ldef, act == 5, 1, node, 0, arena, arena_chunks, h, lane);
            n_sp += __popc(__ballot_sync(0xffffffffu, act == 0));
            n_spp += __popc(__ballot_sync(0xffffffffu, act == 4));
            n_def += __popc(__ballot_sync(0xffffffffu, act == 5));
            const int push = (act == 3) ? nch : 0;
            int pref = push;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                int a = __shfl_up_sync(0xffffffffu, pref, o);
                if (lane >= o) pref += a;
            }
            const int total_push = __shfl_sync(0xffffffffu, pref, 31);
            if (top + total_push > WALK_STACK) { if (lane == 0) atomicOr(&h->status, PETAR_ST_STACK); top = 0; break; }   // cannot happen (throttle above)
            const int at = top + pref - push;
            for (int k = 0; k < push; ++k) stack[at + k] = fc + k;
            top += total_push;
            __syncwarp();
        }
        if (lane == 0) {
            SuperRec* so = &srec[s];
            so->head_sp = lsp.head; so->n_sp = n_sp; so->head_spp = lspp.head; so->n_spp = n_spp;
            so->head_def = ldef.head; so->n_def = n_def;
        }
    }
}

         // > 7 * 21: room for a pure depth-first descent from any state
#define WALK_MIN_CTAS 3
__global__ void __maxnreg__(56) k_walk(DevHeader* __restrict__ h, const NodeW* __restrict__ nw,
                                                          const NodeMac* __restrict__ nmac, GroupRec* __restrict__ grp,
                                                          const SuperRec* __restrict__ srec, const int* __restrict__ smap,
                                                          int* __restrict__ arena, int arena_chunks, double theta, int node_cap,
                                                          long long n_part, int group_cap) {
    __shared__ int s_stack[WALK_WARPS][GWALK_STACK];
    __shared__ float s_lt[PETAR_NLEVELS];          // edge(level) / theta  (inf when theta == 0: nothing is ever "far")
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int* stack = s_stack[w];
    const int ng = h->n_groups;
    if (h->n_nodes > node_cap || h->n_nodes <= 0) return;
    const double twoh = 2.0 * h->h;
    const double rcx = h->c[0], rcy = h->c[1], rcz = h->c[2];
    if (threadIdx.x < PETAR_NLEVELS) s_lt[threadIdx.x] = (theta > 0.0) ? (float)(ldexp(twoh, -(int)threadIdx.x) / theta) : INFINITY;
    __syncthreads();
    unsigned long long t_epep = 0, t_epsp = 0, t_near = 0, t_eplist = 0, t_splist = 0, t_common = 0;
    for (;;) {
        int g = 0;
        if (lane == 0) g = atomicAdd(&h->group_ticket, 1);
        g = __shfl_sync(0xffffffffu, g, 0);
        if (g >= ng) break;
        const GroupRec* gr = &grp[g];
        const int n_i = gr->end - gr->begin;
        // fp32 copy of the group's box (relative to the root centre) and its error bound
        const float fl0 = (float)(gr->lo[0] - rcx), fl1 = (float)(gr->lo[1] - rcy), fl2 = (float)(gr->lo[2] - rcz);
        const float fh0 = (float)(gr->hi[0] - rcx), fh1 = (float)(gr->hi[1] - rcy), fh2 = (float)(gr->hi[2] - rcz);
        const float frm = (float)gr->rmax;
        const float geps = 4.8e-7f * fmaxf(fmaxf(fmaxf(fabsf(fl0), fabsf(fh0)), fmaxf(fabsf(fl1), fabsf(fh1))), fmaxf(fabsf(fl2), fabsf(fh2)));
        ListCursor lsp = {-1, -1, 0, 0}, lspp = {-1, -1, 0, 0}, lepn = {-1, -1, 0, 0}, lepf = {-1, -1, 0, 0};
        int n_sp = 0, n_spp = 0, n_epn = 0, n_epf = 0, n_ep_part = 0, n_epn_part = 0;
        // cells closer to the group's box than the box's longest edge go to the "precise" list: the force
        // kernel evaluates them with float-float coordinates, all others with group-relative floats
        const float gedge = fmaxf(fh0 - fl0, fmaxf(fh1 - fl1, fh2 - fl2));
        const float gedge2 = gedge * gedge;
        // the walk starts from the cells the super-group's walk deferred (k_walk_super), fed in batches
        int sid[PETAR_NSUP];
#pragma unroll
        for (int l = 0; l < PETAR_NSUP; ++l) sid[l] = smap[(size_t)l * n_part + gr->begin];
        const SuperRec* sr = &srec[(size_t)(PETAR_NSUP - 1) * group_cap + sid[PETAR_NSUP - 1]];
        int dchunk = sr->head_def, dremaining = sr->n_def, doff = 0;
        int top = 0;
        // The loop is software-pipelined: the records of the NEXT batch of nodes are requested right after the
        // current batch's children are pushed, so their latency is covered by the list output of the current batch.
        int p = 0, node = -1;
        NodeW c;
        auto pop = [&]() {
            p = 0; node = -1;
            if (top == 0) {                    // frontier empty: take the next (up to 256) deferred cells
                if (dremaining <= 0 || dchunk < 0) return;      // done (or truncated list: arena exhausted, PETAR_ST_LIST_CAP is set)
                const int* cp = arena + (size_t)dchunk * PETAR_CHUNK;
                const int k = min(256, min(dremaining, PETAR_CHUNK_PAYLOAD - doff));
                for (int e = lane; e < k; e += 32) stack[e] = cp[PETAR_CHUNK_HDR + doff + e];
                top = k; dremaining -= k; doff += k;
                if (dremaining > 0 && doff >= PETAR_CHUNK_PAYLOAD) { dchunk = cp[0]; doff = 0; }
                __syncwarp();
            }
            // pop up to 32 nodes; throttle towards depth-first order when the frontier nears its capacity
            // (a pure depth-first descent adds at most 7 entries per level, < WALK_RESERVE in total)
            p = min(32, top);
            if (top + 7 * p > GWALK_STACK - WALK_RESERVE) p = max(1, min(p, (GWALK_STACK - WALK_RESERVE - top) / 7));
            if (lane < p) node = stack[top - p + lane];
            top -= p;
            __syncwarp();
            if (node >= 0) c = nw[node];
        };
        pop();
        while (p > 0) {
            int act = -1;                      // 0 SP, 1 EP near, 2 EP far, 3 open, 4 SP (precise list)
            int nb = 0, ne = 0, fc = 0, nch = 0;
            const int node_cur = node;
            if (node >= 0) {
                const int meta = c.d.w;
                const int level = meta & 255;
                const bool leaf = (meta >> 16) & 1;
                nb = c.d.x; ne = c.d.y; fc = c.d.z; nch = (meta >> 8) & 15;
                // ---- fp32 pre-test with error band --------------------------------------------------------
                const float gx = fmaxf(0.f, fmaxf(c.a.x - fh0, fl0 - c.a.w));
                const float gy = fmaxf(0.f, fmaxf(c.a.y - fh1, fl1 - c.b.x));
                const float gz = fmaxf(0.f, fmaxf(c.a.z - fh2, fl2 - c.b.y));
                const float d2b = fmaf(gz, gz, fmaf(gy, gy, gx * gx));
                const float px = fmaxf(0.f, fmaxf(fl0 - c.b.z, c.b.z - fh0));
                const float py = fmaxf(0.f, fmaxf(fl1 - c.b.w, c.b.w - fh1));
                const float pz = fmaxf(0.f, fmaxf(fl2 - c.c.x, c.c.x - fh2));
                const float d2c = fmaf(pz, pz, fmaf(py, py, px * px));
                const float D = geps + c.c.z;
                const float R = fmaxf(frm, c.c.y);
                const float Dr = fmaf(R, 2.4e-7f, D);
                const float Rm = fmaxf(R - Dr, 0.f), Rp = R + Dr;
                const bool near_yes = d2b < Rm * Rm, near_no = d2b > Rp * Rp;
                const float L = s_lt[level];
                const float Dl = fmaf(L, 2.4e-7f, D);
                const float Lm = fmaxf(L - Dl, 0.f), Lp = L + Dl;
                const bool far_yes = d2c > Lp * Lp, far_no = d2c < Lm * Lm;      // L = inf: Lp*Lp = inf, never far
                if (near_no && far_yes) act = 0;
                else if (!leaf && (near_yes || far_no)) act = 3;
                else if (leaf && near_yes) act = 1;
                else if (leaf && near_no && far_no) act = 2;
                else act = mac_exact(&nmac[node], level, leaf, gr, theta, twoh);
                if (act == 0 && d2b < gedge2) act = 4;
            }
            // children of the opened cells go to the frontier
            const int push = (act == 3) ? nch : 0;
            int pref = push;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                int a = __shfl_up_sync(0xffffffffu, pref, o);
                if (lane >= o) pref += a;
            }
            const int total_push = __shfl_sync(0xffffffffu, pref, 31);
            if (top + total_push > GWALK_STACK) {                 // cannot happen (see the throttle above)
                if (lane == 0) atomicOr(&h->status, PETAR_ST_STACK);
                top = 0;
                break;
            }
            const int at = top + pref - push;
            for (int k = 0; k < push; ++k) stack[at + k] = fc + k;
            top += total_push;
            __syncwarp();
            pop();                             // next batch: its loads overlap the output below
            // outputs of the current batch
            // far leaves: the lanes hold the nodes in frontier order, i.e. siblings in ascending order, so neighbouring lanes often hold
            // leaves whose particle ranges are contiguous; such runs are written as ONE range (EP(g) is a set of particles, rule O7;
            // the force kernel's range expansion gets ~3 x fewer entries)
            const int prev_ne = __shfl_up_sync(0xffffffffu, ne, 1), prev_act = __shfl_up_sync(0xffffffffu, act, 1);
            const bool cont = act == 2 && lane > 0 && prev_act == 2 && prev_ne == nb;
            const unsigned cm = __ballot_sync(0xffffffffu, cont);
            const bool head = act == 2 && !cont;
            const unsigned after = lane < 31 ? (cm >> (lane + 1)) : 0u;
            const int run = __ffs(~after) - 1;                         // lanes that continue my range
            const int ne_run = __shfl_sync(0xffffffffu, ne, min(lane + run, 31));
            // the four lists of the batch.  Usual case: every list has room in its current chunk -- one set of ballots, no per-list
            // branching; otherwise (a new chunk is needed somewhere, about once in 16 batches) the general append, list by list
            const unsigned m_sp = __ballot_sync(0xffffffffu, act == 0), m_spp = __ballot_sync(0xffffffffu, act == 4);
            const unsigned m_epn = __ballot_sync(0xffffffffu, act == 1), m_epf = __ballot_sync(0xffffffffu, head);
            const int c_sp = __popc(m_sp), c_spp = __popc(m_spp), c_epn = __popc(m_epn), c_epf = __popc(m_epf);
            const bool fits = (c_sp == 0 || (lsp.chunk >= 0 && !lsp.dead && lsp.pos + c_sp <= PETAR_CHUNK_PAYLOAD)) &&
                              (c_spp == 0 || (lspp.chunk >= 0 && !lspp.dead && lspp.pos + c_spp <= PETAR_CHUNK_PAYLOAD)) &&
                              (c_epn == 0 || (lepn.chunk >= 0 && !lepn.dead && lepn.pos + 2 * c_epn <= PETAR_CHUNK_PAYLOAD)) &&
                              (c_epf == 0 || (lepf.chunk >= 0 && !lepf.dead && lepf.pos + 2 * c_epf <= PETAR_CHUNK_PAYLOAD));
            if (fits) {
                const unsigned lt = (1u << lane) - 1u;
                if (act == 0) arena[(size_t)lsp.chunk * PETAR_CHUNK + PETAR_CHUNK_HDR + lsp.pos + __popc(m_sp & lt)] = node_cur;
                else if (act == 4) arena[(size_t)lspp.chunk * PETAR_CHUNK + PETAR_CHUNK_HDR + lspp.pos + __popc(m_spp & lt)] = node_cur;
                else if (act == 1) { int* q = arena + (size_t)lepn.chunk * PETAR_CHUNK + PETAR_CHUNK_HDR + lepn.pos + 2 * __popc(m_epn & lt); q[0] = nb; q[1] = ne; }
                else if (head) { int* q = arena + (size_t)lepf.chunk * PETAR_CHUNK + PETAR_CHUNK_HDR + lepf.pos + 2 * __popc(m_epf & lt); q[0] = nb; q[1] = ne_run; }
                lsp.pos += c_sp; lspp.pos += c_spp; lepn.pos += 2 * c_epn; lepf.pos += 2 * c_epf;
            } else {
                list_append(lsp, act == 0, 1, node_cur, 0, arena, arena_chunks, h, lane);
                list_append(lspp, act == 4, 1, node_cur, 0, arena, arena_chunks, h, lane);
                list_append(lepn, act == 1, 2, nb, ne, arena, arena_chunks, h, lane);
                list_append(lepf, head, 2, nb, ne_run, arena, arena_chunks, h, lane);
            }
            n_sp += c_sp; n_spp += c_spp; n_epn += c_epn; n_epf += c_epf;
            const int cn = __reduce_add_sync(0xffffffffu, (act == 1) ? (ne - nb) : 0);
            const int cf = __reduce_add_sync(0xffffffffu, (act == 2) ? (ne - nb) : 0);
            n_epn_part += cn; n_ep_part += cn + cf;
        }
        if (lane == 0) {
            GroupRec* go = &grp[g];
            go->head_sp = lsp.head; go->head_epn = lepn.head; go->head_epf = lepf.head;
            go->n_sp = n_sp; go->n_epn = n_epn; go->n_epf = n_epf;
            go->head_spp = lspp.head; go->n_spp = n_spp;
            go->n_ep_part = n_ep_part; go->n_epn_part = n_epn_part;
#pragma unroll
            for (int l = 0; l < PETAR_NSUP; ++l) go->sid[l] = sid[l];
        }
        int n_common = 0;
#pragma unroll
        for (int l = 0; l < PETAR_NSUP; ++l) { const SuperRec* q = &srec[(size_t)l * group_cap + sid[l]]; n_common += q->n_sp + q->n_spp; }
        t_epep += (unsigned long long)n_i * (unsigned long long)n_ep_part;
        t_near += (unsigned long long)n_i * (unsigned long long)n_epn_part;
        t_epsp += (unsigned long long)n_i * (unsigned long long)(n_sp + n_spp + n_common);
        t_common += (unsigned long long)n_i * (unsigned long long)n_common;
        t_eplist += (unsigned long long)(n_epn + n_epf);
        t_splist += (unsigned long long)(n_sp + n_spp + n_common);
    }
    if (lane == 0) {
        atomicAdd(&h->n_epep, t_epep); atomicAdd(&h->n_epsp, t_epsp); atomicAdd(&h->n_epep_near, t_near);
        atomicAdd(&h->n_ep_list, t_eplist); atomicAdd(&h->n_sp_list, t_splist); atomicAdd(&h->n_epsp_common, t_common);
    }
}

__global__ void k_reset_ticket(DevHeader* h, int which) {
    if (threadIdx.x == 0) { if (which == 0) { h->group_ticket = 0; h->arena_top = 0; for (int l = 0; l < PETAR_NSUP; ++l) { h->n_super[l] = 0; h->super_ticket[l] = 0; } h->n_epep = h->n_epsp = h->n_epep_near = h->n_ep_list = h->n_sp_list = h->n_epsp_common = 0ull; } else h->group_ticket3 = 0; }
}

// the super-group levels (everything the force phase A needs)
cudaError_t launch_walk_supers(petar_tree* t, cudaStream_t s) {
    Workspace& w = t->w;
    stage_begin(t, PETAR_STAGE_WALK_SUPER, s);
    k_reset_ticket<<<1, 32, 0, s>>>(w.hdr, 0);
    KCHECK(s, "k_reset_ticket");
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_walk_super, WALK_WARPS * 32, 0);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    for (int l = 0; l < PETAR_NSUP; ++l) {
        SuperRec* sl = w.srec + (size_t)l * w.group_cap;
        int* ml = w.smap + (size_t)l * t->N;
        k_super_collect<<<cdiv(w.node_cap, 256), 256, 0, s>>>(w.hdr, w.nw, w.key, t->N, sl, w.node_cap, l, PETAR_SUP_LIMIT(l));
        KCHECK(s, "k_super_collect");
        k_super_map<<<t->sm_count * 8, 256, 0, s>>>(w.hdr, sl, ml, l);
        KCHECK(s, "k_super_map");
        k_walk_super<<<t->sm_count * per_sm, WALK_WARPS * 32, 0, s>>>(w.hdr, w.nw, sl, l ? sl - w.group_cap : nullptr, l ? ml - t->N : nullptr,
                                                                     w.arena, w.arena_chunks, t->p.theta, w.node_cap, l);
        KCHECK(s, "k_walk_super");
    }
    petar_count_launch(1 + 3 * PETAR_NSUP);
    stage_end(t, PETAR_STAGE_WALK_SUPER, s);
    return cudaGetLastError();
}

// the per-group walks; ctas_per_sm > 0 limits the grid (tuning experiments)
cudaError_t launch_walk_groups(petar_tree* t, cudaStream_t s, int ctas_per_sm) {
    Workspace& w = t->w;
    stage_begin(t, PETAR_STAGE_WALK, s);
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_walk, WALK_WARPS * 32, 0);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    if (ctas_per_sm > 0 && ctas_per_sm < per_sm) per_sm = ctas_per_sm;
    // the carve-out of the kernels it runs beside (launch_force_units); per device, hence set on every launch
    e = cudaFuncSetAttribute(k_walk, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    k_walk<<<t->sm_count * per_sm, WALK_WARPS * 32, 0, s>>>(w.hdr, w.nw, w.nmac, w.grp, w.srec, w.smap, w.arena, w.arena_chunks, t->p.theta, w.node_cap,
                                                          (long long)t->N, w.group_cap);
    KCHECK(s, "k_walk");
    petar_count_launch(1);
    stage_end(t, PETAR_STAGE_WALK, s);
    return cudaGetLastError();
}

cudaError_t launch_walk(petar_tree* t, cudaStream_t s) {
    cudaError_t e = launch_walk_supers(t, s);
    if (e != cudaSuccess) return e;
    return launch_walk_groups(t, s, 0);
}

// ------------------------------------------------------------------------------------------------
// S9: neighbours.  One warp per group (one CTA for the few groups with a very long near list); lanes own
// i-particles; j runs over the NEAR EP ranges only
// (a leaf that is not near has every pair at r >= R_ij, rule O7), fp64 test of rule O9.
// Pass 1 counts into cnt[original index]; pass 2 (after the scan) fills.
// ------------------------------------------------------------------------------------------------
// Rule O10b: pericentre separation of the pair's Kepler orbit, exactly the operation order of
// DESIGN.md (this file is compiled with -fmad=false; fma only where written).
__device__ __forceinline__ double pericentre(double dx, double dy, double dz, double r2, double wx, double wy, double wz, double mu) {
    const double v2 = fma(wz, wz, fma(wy, wy, wx * wx));
    const double hx = dy * wz - dz * wy, hy = dz * wx - dx * wz, hz = dx * wy - dy * wx;
    const double h2 = fma(hz, hz, fma(hy, hy, hx * hx));
    const double r = sqrt(r2);
    if (r == 0.0) return 0.0;
    const double e2 = v2 - (2.0 * mu) / r;
    double disc = fma(e2, h2, mu * mu);
    if (!(disc > 0.0)) disc = 0.0;
    const double den = mu + sqrt(disc);
    return den > 0.0 ? h2 / den : r;
}

// ORBIT: the two-stage criterion of PAPER.md:346-348 (rule O10c): candidate as in O9 with the Eq. 24 radii,
// kept iff the pair is inside its changeover radius or r_p < C_V min(r_nb,i, r_nb,j).
struct OrbitArgs { const double *vxs, *vys, *vzs, *ms, *routs; double G, Cv; };

struct NbArgs {
    const int* arena; const unsigned* perm;
    const double *xs, *ys, *zs, *rss;
    int* cnt; const long long* offsets; int* indices; long long capacity;
    OrbitArgs oa;
};
struct NbTile { double x[32], y[32], z[32], r[32]; int j[32]; };

// One warp, one block of <= 32 i-particles (lane = particle) of group gr, against the blocks of 32 leaf ranges
// number wsel, wsel + nwarps, ... of the group's near list.  The particles of 32 ranges are flattened (warp scan +
// search), staged 32 at a time in shared memory with one coalesced load per array, then tested by every lane.
// Returns the lane's count; FILL writes the kept neighbours from position o on.
template <bool FILL, bool ORBIT>
__device__ __forceinline__ int nb_sweep(const NbArgs& A, const GroupRec& gr, const int i, const bool vi, const long long o,
                                        const int lane, NbTile& tl, const int wsel, const int nwarps) {
    double xi = 0, yi = 0, zi = 0, ri = 0;
    double vxi = 0, vyi = 0, vzi = 0, mi = 0, roi = 0;
    if (vi) {
        xi = A.xs[i]; yi = A.ys[i]; zi = A.zs[i]; ri = A.rss[i];
        if (ORBIT) { vxi = A.oa.vxs[i]; vyi = A.oa.vys[i]; vzi = A.oa.vzs[i]; mi = A.oa.ms[i]; roi = A.oa.routs[i]; }
    }
    int c = 0, blk = 0;
    int chunk = gr.head_epn;
    int remaining = gr.n_epn * 2;       // entries
    while (chunk >= 0 && remaining > 0) {
        const int* cp = A.arena + (size_t)chunk * PETAR_CHUNK;
        const int ne = min(remaining, PETAR_CHUNK_PAYLOAD);
        for (int e0 = 0; e0 < ne; e0 += 64, ++blk) {
            if (blk % nwarps != wsel) continue;
            int jb_l = 0, cnt_l = 0;
            if (e0 + 2 * lane < ne) { const int2 be = *reinterpret_cast<const int2*>(cp + PETAR_CHUNK_HDR + e0 + 2 * lane); jb_l = be.x; cnt_l = be.y - be.x; }
            int incl = cnt_l;
#pragma unroll
            for (int o2 = 1; o2 < 32; o2 <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, o2); if (lane >= o2) incl += v; }
            const int total = __shfl_sync(0xffffffffu, incl, 31);
            const int excl = incl - cnt_l;
            for (int p0 = 0; p0 < total; p0 += 32) {
                const int p = p0 + lane;
                int lo = 0;                               // smallest range whose inclusive count exceeds p
#pragma unroll
                for (int step = 16; step > 0; step >>= 1) { const int v = __shfl_sync(0xffffffffu, incl, lo + step - 1); if (v <= p) lo += step; }
                lo = min(lo, 31);
                const int rjb = __shfl_sync(0xffffffffu, jb_l, lo), rex = __shfl_sync(0xffffffffu, excl, lo);
                __syncwarp();
                if (p < total) {
                    const int j = rjb + (p - rex);
                    tl.x[lane] = A.xs[j]; tl.y[lane] = A.ys[j]; tl.z[lane] = A.zs[j]; tl.r[lane] = A.rss[j]; tl.j[lane] = j;
                }
                __syncwarp();
                const int nb = min(32, total - p0);
                for (int k = 0; k < nb; ++k) {
                    const int j = tl.j[k];
                    const double xj = tl.x[k], yj = tl.y[k], zj = tl.z[k], rj = tl.r[k];
                    double dx = xi - xj, dy = yi - yj, dz = zi - zj;
                    double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                    double R = fmax(ri, rj);
                    bool keep = vi && j != i && r2 < R * R;
                    if (ORBIT && keep) {
                        const double Ro = fmax(roi, A.oa.routs[j]);
                        if (!(r2 < Ro * Ro)) {
                            const double rp = pericentre(dx, dy, dz, r2, vxi - A.oa.vxs[j], vyi - A.oa.vys[j], vzi - A.oa.vzs[j], A.oa.G * (mi + A.oa.ms[j]));
                            keep = rp < A.oa.Cv * fmin(ri, rj);
                        }
                    }
                    if (keep) {
                        if (FILL) { if (o + c < A.capacity) A.indices[o + c] = (int)A.perm[j]; }
                        ++c;
                    }
                }
            }
        }
        remaining -= ne;
        chunk = cp[0];
    }
    return c;
}

// groups whose near list is long (a massive particle's r_out reaches thousands of others) go to k_neighbors_big
#define NB_BIG_WORK 32768
__device__ __forceinline__ bool nb_is_big(const GroupRec& gr) { return (long long)gr.n_epn_part * (long long)(gr.end - gr.begin) > NB_BIG_WORK; }

// One warp per group.  queue[0] = number of big groups, queue[1..] = their ids (filled by the count pass).
template <bool FILL, bool ORBIT>
__global__ void __launch_bounds__(256) k_neighbors(DevHeader* __restrict__ h, const GroupRec* __restrict__ grp, const NbArgs A, int* __restrict__ queue) {
    __shared__ NbTile s_tile[8];
    const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
    const int ng = h->n_groups;
    for (;;) {
        int g = 0;
        if (lane == 0) g = atomicAdd(&h->group_ticket3, 1);
        g = __shfl_sync(0xffffffffu, g, 0);
        if (g >= ng) break;
        const GroupRec gr = grp[g];
        if (nb_is_big(gr)) {
            if (!FILL && lane == 0) queue[1 + atomicAdd(&queue[0], 1)] = g;
            continue;
        }
        for (int ib = gr.begin; ib < gr.end; ib += 32) {
            const int i = ib + lane;
            const bool vi = i < gr.end;
            unsigned oi = 0;
            long long o = 0;
            if (vi) { oi = A.perm[i]; if (FILL) o = A.offsets[oi]; }
            const int c = nb_sweep<FILL, ORBIT>(A, gr, i, vi, o, lane, s_tile[wp], 0, 1);
            if (!FILL && vi) A.cnt[oi] = c;
        }
    }
}

// One CTA (8 warps) per big group: the warps share out the blocks of 32 leaf ranges.  Every warp counts its share
// first, so the rows are filled at fixed positions (warp 0's neighbours, then warp 1's, ...): deterministic.
template <bool FILL, bool ORBIT>
__global__ void __launch_bounds__(256) k_neighbors_big(const GroupRec* __restrict__ grp, const NbArgs A, const int* __restrict__ queue) {
    __shared__ NbTile s_tile[8];
    __shared__ int s_cnt[8][32];
    const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
    const int nq = queue[0];
    for (int q = blockIdx.x; q < nq; q += gridDim.x) {
        const GroupRec gr = grp[queue[1 + q]];
        for (int ib = gr.begin; ib < gr.end; ib += 32) {
            const int i = ib + lane;
            const bool vi = i < gr.end;
            unsigned oi = 0;
            long long o = 0;
            if (vi) { oi = A.perm[i]; if (FILL) o = A.offsets[oi]; }
            __syncthreads();                                     // s_cnt of the previous block consumed
            s_cnt[wp][lane] = nb_sweep<false, ORBIT>(A, gr, i, vi, 0, lane, s_tile[wp], wp, 8);
            __syncthreads();
            if (FILL) {
                for (int w2 = 0; w2 < wp; ++w2) o += s_cnt[w2][lane];
                nb_sweep<true, ORBIT>(A, gr, i, vi, o, lane, s_tile[wp], wp, 8);
            } else if (wp == 0 && vi) {
                int c = 0;
                for (int w2 = 0; w2 < 8; ++w2) c += s_cnt[w2][lane];
                A.cnt[oi] = c;
            }
        }
    }
}

__global__ void __launch_bounds__(256) k_gather_vel(const unsigned* __restrict__ perm, long long n, const double* __restrict__ vx,
                                                    const double* __restrict__ vy, const double* __restrict__ vz,
                                                    double* __restrict__ vxs, double* __restrict__ vys, double* __restrict__ vzs) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const unsigned o = perm[i];
    vxs[i] = vx[o]; vys[i] = vy[o]; vzs[i] = vz[o];
}

__global__ void k_nb_status(const long long* __restrict__ offsets, long long n, long long capacity, int* __restrict__ status_dev,
                            DevHeader* __restrict__ h, int have_indices) {
    if (threadIdx.x == 0) {
        long long tot = offsets[n];
        h->nb_total = (unsigned long long)tot;
        int over = (have_indices && tot > capacity) ? 1 : 0;
        if (status_dev) *status_dev = over;
        if (over) atomicOr(&h->status, PETAR_ST_NB_CAP);
    }
}

cudaError_t launch_neighbors(petar_tree* t, int64_t* offsets, int32_t* indices, int64_t capacity, int32_t* status_dev, cudaStream_t s,
                             const double* vx, const double* vy, const double* vz, double Cv) {
    Workspace& w = t->w;
    const long long n = t->N;
    const double* rss = t->r_search ? w.rss : w.routs;
    const bool orbit = vx != nullptr;
    NbArgs A = {w.arena, w.idx, w.xs, w.ys, w.zs, rss, w.nb_cnt, nullptr, nullptr, 0, {w.vxs, w.vys, w.vzs, w.ms, w.routs, t->p.G, Cv}};
    stage_begin(t, PETAR_STAGE_NEIGHBOR, s);
    const int grid = t->sm_count * 8, grid_big = t->sm_count;
    if (orbit) {
        k_gather_vel<<<cdiv(n, 256), 256, 0, s>>>(w.idx, n, vx, vy, vz, w.vxs, w.vys, w.vzs);
        KCHECK(s, "k_gather_vel");
        petar_count_launch(1);
    }
    cudaError_t e = cudaSuccess;
    if (orbit || !t->nb_counted) {          // the count pass (two-phase output: a count call followed by a fill call counts once)
        e = cudaMemsetAsync(w.nb_queue, 0, 4, s);
        if (e != cudaSuccess) return e;
        k_reset_ticket<<<1, 32, 0, s>>>(w.hdr, 1);
        KCHECK(s, "k_reset_ticket");
        if (orbit) { k_neighbors<false, true><<<grid, 256, 0, s>>>(w.hdr, w.grp, A, w.nb_queue); k_neighbors_big<false, true><<<grid_big, 256, 0, s>>>(w.grp, A, w.nb_queue); }
        else { k_neighbors<false, false><<<grid, 256, 0, s>>>(w.hdr, w.grp, A, w.nb_queue); k_neighbors_big<false, false><<<grid_big, 256, 0, s>>>(w.grp, A, w.nb_queue); }
        KCHECK(s, "k_neighbors");
        petar_count_launch(3);
        t->nb_counted = !orbit;
    }
    e = launch_scan_i32_to_i64(w.nb_cnt, (long long*)offsets, n, (long long*)w.scan_tmp, s);
    if (e != cudaSuccess) return e;
    if (indices) {
        A.offsets = (const long long*)offsets; A.indices = indices; A.capacity = capacity;
        k_reset_ticket<<<1, 32, 0, s>>>(w.hdr, 1);
        KCHECK(s, "k_reset_ticket");
        if (orbit) { k_neighbors<true, true><<<grid, 256, 0, s>>>(w.hdr, w.grp, A, w.nb_queue); k_neighbors_big<true, true><<<grid_big, 256, 0, s>>>(w.grp, A, w.nb_queue); }
        else { k_neighbors<true, false><<<grid, 256, 0, s>>>(w.hdr, w.grp, A, w.nb_queue); k_neighbors_big<true, false><<<grid_big, 256, 0, s>>>(w.grp, A, w.nb_queue); }
        KCHECK(s, "k_neighbors");
        petar_count_launch(3);
    }
    k_nb_status<<<1, 32, 0, s>>>((const long long*)offsets, n, capacity, status_dev, w.hdr, indices ? 1 : 0);
    KCHECK(s, "k_nb_status");
    petar_count_launch(1);
    stage_end(t, PETAR_STAGE_NEIGHBOR, s);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// list export (tests): flatten the chunk chains.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int common_cells(const GroupRec* gr, const SuperRec* __restrict__ srec, int group_cap) {
    int c = 0;
    for (int l = 0; l < PETAR_NSUP; ++l) { const SuperRec* q = &srec[(size_t)l * group_cap + gr->sid[l]]; c += q->n_sp + q->n_spp; }
    return c;
}
__global__ void k_list_sizes(const DevHeader* __restrict__ h, const GroupRec* __restrict__ grp, const SuperRec* __restrict__ srec, int group_cap, int* __restrict__ sizes) {
    int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= h->n_groups) return;
    sizes[3 * g] = grp[g].n_sp + grp[g].n_spp + common_cells(&grp[g], srec, group_cap); sizes[3 * g + 1] = 2 * grp[g].n_epn; sizes[3 * g + 2] = 2 * grp[g].n_epf;
}
__global__ void k_list_flatten(const DevHeader* __restrict__ h, const GroupRec* __restrict__ grp, const SuperRec* __restrict__ srec, int group_cap, const int* __restrict__ arena,
                               const long long* __restrict__ offs, int* __restrict__ out, long long out_entries) {
    const int lane = threadIdx.x & 31;
    long long wid = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (wid >= 3ll * h->n_groups) return;
    int g = (int)(wid / 3), which = (int)(wid % 3);
    int chunk = which == 0 ? grp[g].head_sp : which == 1 ? grp[g].head_epn : grp[g].head_epf;
    int remaining = which == 0 ? grp[g].n_sp : which == 1 ? 2 * grp[g].n_epn : 2 * grp[g].n_epf;
    long long o = offs[wid];
    for (int part = 0; part < 2 + 2 * PETAR_NSUP; ++part) {
        while (chunk >= 0 && remaining > 0) {
            const int* cp = arena + (size_t)chunk * PETAR_CHUNK;
            int ne = min(remaining, PETAR_CHUNK_PAYLOAD);
            for (int e = lane; e < ne; e += 32) if (o + e < out_entries) out[o + e] = cp[PETAR_CHUNK_HDR + e];
            o += ne; remaining -= ne; chunk = cp[0];
        }
        if (which != 0) break;
        // "SP" = own plain cells, own precise cells, then every level's common cells (plain, precise)
        if (part == 0) { chunk = grp[g].head_spp; remaining = grp[g].n_spp; }
        else if (part < 1 + 2 * PETAR_NSUP) {
            const SuperRec* sr = &srec[(size_t)((part - 1) >> 1) * group_cap + grp[g].sid[(part - 1) >> 1]];
            if ((part - 1) & 1) { chunk = sr->head_spp; remaining = sr->n_spp; } else { chunk = sr->head_sp; remaining = sr->n_sp; }
        }
    }
}
__global__ void k_group_cnt(const DevHeader* __restrict__ h, const GroupRec* __restrict__ grp, const SuperRec* __restrict__ srec, int group_cap, int* __restrict__ out, int what, int walked) {
    int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= h->n_groups) return;
    if (what == PETAR_DBG_GROUP_CNT) { out[4 * g] = grp[g].n_sp + grp[g].n_spp + (walked ? common_cells(&grp[g], srec, group_cap) : 0); out[4 * g + 1] = grp[g].n_epn; out[4 * g + 2] = grp[g].n_epf; out[4 * g + 3] = grp[g].n_ep_part; }
    else if (what == PETAR_DBG_GROUP_SUPER) {
        for (int l = 0; l < 2; ++l) {
            const int ll = l < PETAR_NSUP ? l : PETAR_NSUP - 1;
            const SuperRec* sr = &srec[(size_t)ll * group_cap + grp[g].sid[ll]];
            out[8 * g + 4 * l] = grp[g].sid[ll]; out[8 * g + 4 * l + 1] = sr->end - sr->begin; out[8 * g + 4 * l + 2] = sr->n_sp + sr->n_spp; out[8 * g + 4 * l + 3] = sr->n_def;
        }
    }
    else { out[2 * g] = grp[g].begin; out[2 * g + 1] = grp[g].end; }
}
__global__ void k_group_dbl(const DevHeader* __restrict__ h, const GroupRec* __restrict__ grp, double* __restrict__ out) {
    int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= h->n_groups) return;
    for (int k = 0; k < 3; ++k) { out[7 * g + k] = grp[g].lo[k]; out[7 * g + 3 + k] = grp[g].hi[k]; }
    out[7 * g + 6] = grp[g].rmax;
}
__global__ void k_node_dbl(const DevHeader* __restrict__ h, const NodeMac* __restrict__ nmac, const NodeMom* __restrict__ nmom, double* __restrict__ out) {
    int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= h->n_nodes) return;
    double* D = out + 17ll * n;
    D[0] = nmom[n].M;
    for (int k = 0; k < 3; ++k) { D[1 + k] = nmac[n].com[k]; D[4 + k] = nmac[n].lo[k]; D[7 + k] = nmac[n].hi[k]; }
    D[10] = nmac[n].rmax;
    for (int k = 0; k < 6; ++k) D[11 + k] = nmom[n].Q[k];
}

// n_groups / n_nodes are passed by the caller (api.cu reads the header back first)
cudaError_t launch_export_lists(petar_tree* t, int what, void* dst, size_t dst_bytes, cudaStream_t s) {
    Workspace& w = t->w;
    int ng = t->h_groups, nn = t->h_nodes;
    if (what == PETAR_DBG_GROUP_CNT || what == PETAR_DBG_GROUP_INT || what == PETAR_DBG_GROUP_SUPER) {
        size_t need = (size_t)ng * (what == PETAR_DBG_GROUP_INT ? 8 : what == PETAR_DBG_GROUP_SUPER ? 32 : 16);
        if (dst_bytes < need) return cudaErrorInvalidValue;
        if (ng) k_group_cnt<<<cdiv(ng, 256), 256, 0, s>>>(w.hdr, w.grp, w.srec, w.group_cap, (int*)dst, what, t->walked ? 1 : 0);
        KCHECK(s, "k_group_cnt");
    } else if (what == PETAR_DBG_GROUP_DBL) {
        if (dst_bytes < (size_t)ng * 56) return cudaErrorInvalidValue;
        if (ng) k_group_dbl<<<cdiv(ng, 256), 256, 0, s>>>(w.hdr, w.grp, (double*)dst);
        KCHECK(s, "k_group_dbl");
    } else if (what == PETAR_DBG_NODE_DBL) {
        if (dst_bytes < (size_t)nn * 136) return cudaErrorInvalidValue;
        if (nn) k_node_dbl<<<cdiv(nn, 256), 256, 0, s>>>(w.hdr, w.nmac, w.nmom, (double*)dst);
        KCHECK(s, "k_node_dbl");
    } else if (what == PETAR_DBG_LIST_OFFS || what == PETAR_DBG_LISTS) {
        // sizes -> scan -> flatten
        if (!ng) return cudaSuccess;
        int* sizes = w.exp_scratch;                                       // 3 ng ints
        long long* offs = (long long*)(w.exp_scratch + 4ll * (ng + 1));   // 3 ng + 1 int64 (16-byte aligned)
        k_list_sizes<<<cdiv(ng, 256), 256, 0, s>>>(w.hdr, w.grp, w.srec, w.group_cap, sizes);
        KCHECK(s, "k_list_sizes");
        cudaError_t e = launch_scan_i32_to_i64(sizes, offs, 3ll * ng, (long long*)w.scan_tmp, s);
        if (e != cudaSuccess) return e;
        if (what == PETAR_DBG_LIST_OFFS) {
            if (dst_bytes < (size_t)(3ll * ng + 1) * 8) return cudaErrorInvalidValue;
            return cudaMemcpyAsync(dst, offs, (size_t)(3ll * ng + 1) * 8, cudaMemcpyDeviceToDevice, s);
        }
        k_list_flatten<<<cdiv(3ll * ng * 32, 256), 256, 0, s>>>(w.hdr, w.grp, w.srec, w.group_cap, w.arena, offs, (int*)dst, (long long)(dst_bytes / 4));
        KCHECK(s, "k_list_flatten");
    }
    return cudaGetLastError();
}

// build.cu -- steps S0-S6: bounding cube, Morton keys, stable LSD radix sort, sorted SoA gather,
// octree from sorted keys (no level loop: nodes are enumerated per key boundary), bottom-up
// moments, i-groups.   Compiled with -fmad=false: every fp64 operation below is exactly the one
// written (fma only where rule O5 says so), because key, permutation, node and group tables must be
// bit-identical to an independent fp64 implementation of DESIGN.md's rules O1-O6.
#include <cooperative_groups.h>
#include "internal.cuh"
namespace cg = cooperative_groups;

// ------------------------------------------------------------------------------------------------
// small device helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long enc_f64(double d) {
    unsigned long long b = (unsigned long long)__double_as_longlong(d);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double dec_f64(unsigned long long e) {
    unsigned long long b = (e >> 63) ? (e & 0x7fffffffffffffffull) : ~e;
    return __longlong_as_double((long long)b);
}
__device__ __forceinline__ unsigned long long spread21(unsigned long long x) {
    x &= 0x1fffffull;
    x = (x | x << 32) & 0x1f00000000ffffull;
    x = (x | x << 16) & 0x1f0000ff0000ffull;
    x = (x | x << 8) & 0x100f00f00f00f00full;
    x = (x | x << 4) & 0x10c30c30c30c30c3ull;
    x = (x | x << 2) & 0x1249249249249249ull;
    return x;
}
__device__ __forceinline__ unsigned compact21(unsigned long long x) {   // inverse of spread21
    x &= 0x1249249249249249ull;
    x = (x | x >> 2) & 0x10c30c30c30c30c3ull;
    x = (x | x >> 4) & 0x100f00f00f00f00full;
    x = (x | x >> 8) & 0x1f0000ff0000ffull;
    x = (x | x >> 16) & 0x1f00000000ffffull;
    x = (x | x >> 32) & 0x1fffffull;
    return (unsigned)x;
}

// ------------------------------------------------------------------------------------------------
// S0: header reset + bounding box
// ------------------------------------------------------------------------------------------------
__global__ void k_reset_header(DevHeader* h) {
    if (threadIdx.x == 0) {
        for (int k = 0; k < 3; ++k) { h->bbox[k] = ~0ull; h->bbox[3 + k] = 0ull; }
        h->n_nodes = 0; h->n_groups = 0; h->status = 0; h->arena_top = 0;
        h->group_ticket = 0; h->group_ticket2 = 0; h->group_ticket3 = 0; for (int l = 0; l < PETAR_NSUP; ++l) { h->n_super[l] = 0; h->super_ticket[l] = 0; }
        h->n_epep = h->n_epsp = h->n_epep_near = h->n_ep_list = h->n_sp_list = h->n_epsp_common = 0ull; h->nb_total = 0ull;
        for (int l = 0; l < PETAR_NLEVELS + 2; ++l) h->level_off[l] = 0;
        h->rank_done = 0;
    }
}

__global__ void __launch_bounds__(256) k_bbox(const double* __restrict__ x, const double* __restrict__ y,
                                              const double* __restrict__ z, long long n, DevHeader* h) {
    double lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    bool bad = false;
    // two particles per iteration with 16-byte loads when the arrays are 16-byte aligned (torch allocations are)
    const bool vec = ((((uintptr_t)x) | ((uintptr_t)y) | ((uintptr_t)z)) & 15u) == 0;
    const long long n2 = vec ? n / 2 : 0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n2; i += stride) {
        const double2 vx = reinterpret_cast<const double2*>(x)[i], vy = reinterpret_cast<const double2*>(y)[i], vz = reinterpret_cast<const double2*>(z)[i];
        bad |= !(isfinite(vx.x) && isfinite(vx.y) && isfinite(vy.x) && isfinite(vy.y) && isfinite(vz.x) && isfinite(vz.y));
        lo[0] = fmin(lo[0], fmin(vx.x, vx.y)); hi[0] = fmax(hi[0], fmax(vx.x, vx.y));
        lo[1] = fmin(lo[1], fmin(vy.x, vy.y)); hi[1] = fmax(hi[1], fmax(vy.x, vy.y));
        lo[2] = fmin(lo[2], fmin(vz.x, vz.y)); hi[2] = fmax(hi[2], fmax(vz.x, vz.y));
    }
    for (long long i = 2 * n2 + blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += stride) {
        const double v[3] = {x[i], y[i], z[i]};
        bad |= !(isfinite(v[0]) && isfinite(v[1]) && isfinite(v[2]));
#pragma unroll
        for (int k = 0; k < 3; ++k) { lo[k] = fmin(lo[k], v[k]); hi[k] = fmax(hi[k], v[k]); }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k)
        for (int o = 16; o; o >>= 1) {
            lo[k] = fmin(lo[k], __shfl_xor_sync(0xffffffffu, lo[k], o));
            hi[k] = fmax(hi[k], __shfl_xor_sync(0xffffffffu, hi[k], o));
        }
    bad = __any_sync(0xffffffffu, bad);
    if ((threadIdx.x & 31) == 0) {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            if (lo[k] <= hi[k]) { atomicMin(&h->bbox[k], enc_f64(lo[k])); atomicMax(&h->bbox[3 + k], enc_f64(hi[k])); }
        }
        if (bad) atomicOr(&h->status, PETAR_ST_NONFINITE);
    }
}

// O1: root cube.  c = 0.5 (lo + hi); L = max extent; v = 0.5 L (1 + 2^-20); h = 2^e with frexp(v) = (f, e).
__global__ void k_root(DevHeader* h) {
    if (threadIdx.x != 0) return;
    double L = 0.0;
    for (int k = 0; k < 3; ++k) {
        double lo = dec_f64(h->bbox[k]), hi = dec_f64(h->bbox[3 + k]);
        h->c[k] = 0.5 * (lo + hi);
        double e = hi - lo;
        if (e > L) L = e;
    }
    double hh;
    if (!(L > 0.0) || !isfinite(L)) hh = 1.0;
    else {
        double v = 0.5 * L * (1.0 + 9.5367431640625e-07);   // 2^-20
        int e; (void)frexp(v, &e);
        hh = ldexp(1.0, e);
    }
    h->h = hh;
    for (int k = 0; k < 3; ++k) h->o[k] = h->c[k] - hh;
    h->inv_s = ldexp(1.0, PETAR_MAXLEVEL) / (2.0 * hh);     // exact: power of two
}

// O2 + O3: keys.  Two particles per thread (16-byte loads and stores when the input arrays are 16-byte aligned).
__device__ __forceinline__ unsigned long long morton_key(const double vx, const double vy, const double vz, const double o0, const double o1,
                                                         const double o2, const double inv_s) {
    const double v[3] = {vx, vy, vz}, o[3] = {o0, o1, o2};
    unsigned long long q[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const double g = floor((v[k] - o[k]) * inv_s);
        const long long qi = (g >= 0.0) ? ((g < 2097152.0) ? (long long)g : 2097151ll) : 0ll;   // NaN -> 0
        q[k] = (unsigned long long)qi;
    }
    return (spread21(q[0]) << 2) | (spread21(q[1]) << 1) | spread21(q[2]);
}
// Also packs the particle's inputs into one 64-byte record (x, y, z, m, r_out, r_search, -, -) in the caller's order: the
// gather by the sorted permutation then fetches ONE aligned 64-byte record per particle instead of five or six scattered
// 8-byte values, each of which costs a 64-128-byte DRAM fetch (profiles/hbm_r02_config5.md: 604 -> ~140 bytes moved per particle).
__global__ void __launch_bounds__(256) k_keys(const double* __restrict__ x, const double* __restrict__ y,
                                              const double* __restrict__ z, const double* __restrict__ m, const double* __restrict__ ro,
                                              const double* __restrict__ rs, long long n, const DevHeader* __restrict__ h,
                                              unsigned long long* __restrict__ key, unsigned* __restrict__ idx, double2* __restrict__ rec) {
    const long long i = 2 * (blockIdx.x * (long long)blockDim.x + threadIdx.x);
    if (i >= n) return;
    const double inv_s = h->inv_s, o0 = h->o[0], o1 = h->o[1], o2 = h->o[2];
    const bool vec = ((((uintptr_t)x) | ((uintptr_t)y) | ((uintptr_t)z) | ((uintptr_t)m) | ((uintptr_t)ro) | ((uintptr_t)rs)) & 15u) == 0;
    if (vec && i + 1 < n) {
        const double2 vx = *reinterpret_cast<const double2*>(x + i), vy = *reinterpret_cast<const double2*>(y + i), vz = *reinterpret_cast<const double2*>(z + i);
        const double2 vm = *reinterpret_cast<const double2*>(m + i), vr = *reinterpret_cast<const double2*>(ro + i);
        const double2 vs = rs ? *reinterpret_cast<const double2*>(rs + i) : vr;
        ulonglong2 k2;
        k2.x = morton_key(vx.x, vy.x, vz.x, o0, o1, o2, inv_s); k2.y = morton_key(vx.y, vy.y, vz.y, o0, o1, o2, inv_s);
        *reinterpret_cast<ulonglong2*>(key + i) = k2;
        *reinterpret_cast<uint2*>(idx + i) = make_uint2((unsigned)i, (unsigned)i + 1u);
        double2* r = rec + 4 * i;
        r[0] = make_double2(vx.x, vy.x); r[1] = make_double2(vz.x, vm.x); r[2] = make_double2(vr.x, vs.x); r[3] = make_double2(0.0, 0.0);
        r[4] = make_double2(vx.y, vy.y); r[5] = make_double2(vz.y, vm.y); r[6] = make_double2(vr.y, vs.y); r[7] = make_double2(0.0, 0.0);
    } else {
        for (long long j = i; j < min(i + 2, n); ++j) {
            key[j] = morton_key(x[j], y[j], z[j], o0, o1, o2, inv_s); idx[j] = (unsigned)j;
            double2* r = rec + 4 * j;
            const double vr = ro[j];
            r[0] = make_double2(x[j], y[j]); r[1] = make_double2(z[j], m[j]); r[2] = make_double2(vr, rs ? rs[j] : vr); r[3] = make_double2(0.0, 0.0);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// S2: stable LSD radix sort of (key, idx), 8 passes x 8 bits.  Tile = 2048 elements per CTA.
// ------------------------------------------------------------------------------------------------
#define SORT_TILE 2048
#define SORT_THREADS 256
#define SORT_ITEMS 8

// per-block digit counts of the current pass:  blk[d * nblk + b]
__global__ void __launch_bounds__(SORT_THREADS) k_sort_count(const unsigned long long* __restrict__ key, long long n, int shift,
                                                             unsigned* __restrict__ blk, int nblk, unsigned* __restrict__ tot) {
    __shared__ unsigned cnt[256];
    cnt[threadIdx.x] = 0;
    __syncthreads();
    long long base = (long long)blockIdx.x * SORT_TILE;
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        long long i = base + r * SORT_THREADS + threadIdx.x;
        if (i < n) atomicAdd(&cnt[(unsigned)(key[i] >> shift) & 255u], 1u);
    }
    __syncthreads();
    blk[threadIdx.x * nblk + blockIdx.x] = cnt[threadIdx.x];
    if (cnt[threadIdx.x]) atomicAdd(&tot[threadIdx.x], cnt[threadIdx.x]);      // digit totals of this pass
}

// one CTA per digit d: blk[d][b] <- (number of keys with smaller digit) + (same digit in earlier blocks)
__global__ void __launch_bounds__(256) k_sort_scan(unsigned* __restrict__ blk, int nblk, const unsigned* __restrict__ tot) {
    __shared__ unsigned red[256];
    __shared__ unsigned carry_s;
    const int d = blockIdx.x, t = threadIdx.x;
    // total of every digit e < d (from the pass's digit totals; the rows of other digits are being
    // rewritten concurrently by their own CTAs and must not be read here)
    red[t] = (t < d) ? tot[t] : 0u;
    __syncthreads();
    for (int o = 128; o; o >>= 1) { if (t < o) red[t] += red[t + o]; __syncthreads(); }
    if (t == 0) carry_s = red[0];
    __syncthreads();
    unsigned* row = blk + (size_t)d * nblk;
    for (int b0 = 0; b0 < nblk; b0 += 256) {
        int b = b0 + t;
        unsigned v = (b < nblk) ? row[b] : 0u;
        // block inclusive scan (Hillis-Steele in smem)
        __syncthreads();
        red[t] = v;
        __syncthreads();
        for (int o = 1; o < 256; o <<= 1) {
            unsigned a = (t >= o) ? red[t - o] : 0u;
            __syncthreads();
            red[t] += a;
            __syncthreads();
        }
        unsigned incl = red[t], carry = carry_s;
        if (b < nblk) row[b] = carry + incl - v;
        __syncthreads();
        if (t == 255) carry_s = carry + incl;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(SORT_THREADS) k_sort_scatter(const unsigned long long* __restrict__ kin, const unsigned* __restrict__ vin,
                                                               unsigned long long* __restrict__ kout, unsigned* __restrict__ vout,
                                                               const unsigned* __restrict__ blk, int nblk, long long n, int shift) {
    __shared__ unsigned wcnt[SORT_THREADS / 32][256];
    const int t = threadIdx.x, lane = t & 31, w = t >> 5;
    for (int k = t; k < (SORT_THREADS / 32) * 256; k += SORT_THREADS) (&wcnt[0][0])[k] = 0;
    __syncthreads();
    const long long base = (long long)blockIdx.x * SORT_TILE + (long long)w * (SORT_TILE / (SORT_THREADS / 32));
    unsigned long long k[SORT_ITEMS];
    unsigned v[SORT_ITEMS], rank[SORT_ITEMS];
    const unsigned lt = (1u << lane) - 1u;
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        long long i = base + r * 32 + lane;
        bool ok = i < n;
        k[r] = ok ? kin[i] : ~0ull;
        v[r] = ok ? vin[i] : 0u;
        unsigned d = ok ? ((unsigned)(k[r] >> shift) & 255u) : 255u;
        unsigned peers = __match_any_sync(0xffffffffu, d);
        int leader = __ffs(peers) - 1;
        unsigned prev = 0;
        if (lane == leader) { prev = wcnt[w][d]; wcnt[w][d] = prev + __popc(peers); }
        prev = __shfl_sync(0xffffffffu, prev, leader);
        rank[r] = prev + __popc(peers & lt);
        __syncwarp();
    }
    __syncthreads();
    {   // per digit (thread t = digit): exclusive scan over warps, seeded with the global block offset
        unsigned run = blk[(size_t)t * nblk + blockIdx.x];
#pragma unroll
        for (int ww = 0; ww < SORT_THREADS / 32; ++ww) { unsigned c = wcnt[ww][t]; wcnt[ww][t] = run; run += c; }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        long long i = base + r * 32 + lane;
        if (i < n) {
            unsigned d = (unsigned)(k[r] >> shift) & 255u;
            unsigned pos = wcnt[w][d] + rank[r];
            kout[pos] = k[r];
            vout[pos] = v[r];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// S3: gather into sorted order + fp32 float-float records relative to the root centre
// ------------------------------------------------------------------------------------------------
// One sorted position per thread: its 64-byte input record (packed by k_keys) is fetched with four 16-byte loads.  Also the
// finiteness / sign checks of m, r_out, r_search (the positions were checked by k_bbox).
__global__ void __launch_bounds__(256) k_gather(const unsigned* __restrict__ idx, long long n, DevHeader* __restrict__ h,
                                                const double2* __restrict__ rec, const bool have_rs,
                                                double* __restrict__ xs, double* __restrict__ ys, double* __restrict__ zs,
                                                double* __restrict__ ms, double* __restrict__ ros, double* __restrict__ rss,
                                                float4* __restrict__ pa, float4* __restrict__ pb) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    bool bad = false;
    if (i < n) {
        const double2* r = rec + 4 * (size_t)idx[i];
        const double2 r0 = r[0], r1 = r[1], r2 = r[2];
        const double vx = r0.x, vy = r0.y, vz = r1.x, vm = r1.y, vr = r2.x, vq = r2.y;
        bad = !(isfinite(vm) && isfinite(vr) && vr > 0.0);
        xs[i] = vx; ys[i] = vy; zs[i] = vz; ms[i] = vm; ros[i] = vr;
        if (have_rs) { rss[i] = vq; bad |= !(isfinite(vq) && vq >= vr); }
        const double dx = vx - h->c[0], dy = vy - h->c[1], dz = vz - h->c[2];
        const float xh = (float)dx, yh = (float)dy, zh = (float)dz;
        const float xl = (float)(dx - (double)xh), yl = (float)(dy - (double)yh), zl = (float)(dz - (double)zh);
        pa[i] = make_float4(xh, yh, zh, (float)vm);
        pb[i] = make_float4(xl, yl, zl, (float)(1.0 / vr));
    }
    if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) atomicOr(&h->status, PETAR_ST_NONFINITE);
}

// ------------------------------------------------------------------------------------------------
// S4: octree from sorted keys.
//   D[i]  (i = 0..N) = number of leading octal digits keys i-1 and i share (-1 at both array ends).
//   Keys i-1 and i lie in the same level-l cell iff D[i] >= l.
//   depth[i]  = leaf level of particle i  = smallest l whose cell holds <= n_leaf particles (cap 21)
//   glevel[i] = group level               = same with n_group, capped by depth
//   A level-l node starts at boundary i  iff  D[i] < l <= depth[i].
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_diverge(const unsigned long long* __restrict__ key, long long n, signed char* __restrict__ D) {
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i > n) return;
    int d = -1;
    if (i > 0 && i < n) {
        unsigned long long xr = key[i - 1] ^ key[i];
        d = xr ? (__clzll((long long)xr) - 1) / 3 : PETAR_MAXLEVEL;     // bit 62 is the top key bit
    }
    D[i] = (signed char)d;
}

// smallest level l such that the level-l cell containing particle i holds <= L particles, using the
// window D[i-L+1 .. i+L] held in shared memory `sd` (index 0 <-> boundary `w0`).  Returns up to 22
// (22 = even the level-21 cell is over-full).
__device__ __forceinline__ int level_for_limit(const signed char* sd, long long w0, long long i, long long n, int L) {
    int best = 127, run = 127;
    for (int k = 1; k <= L; ++k) {
        long long e = i + k;
        int de = (e <= n) ? (int)sd[e - w0] : -1;
        run = min(run, de);
        long long b = i - L + k;
        if (b >= 0) best = min(best, max((int)sd[b - w0], run));
    }
    return best + 1;
}

#define DEPTH_THREADS 256
__global__ void __launch_bounds__(DEPTH_THREADS) k_depth(const unsigned long long* __restrict__ key, const signed char* __restrict__ D,
                                                         long long n, int n_leaf, int n_group,
                                                         signed char* __restrict__ depth, signed char* __restrict__ glevel,
                                                         int* __restrict__ gflag) {
    extern __shared__ signed char sd[];
    const long long i0 = (long long)blockIdx.x * DEPTH_THREADS;
    const int halo = n_group;
    const long long w0 = i0 - halo;
    const int wn = DEPTH_THREADS + 2 * halo + 1;
    for (int k = threadIdx.x; k < wn; k += DEPTH_THREADS) {
        long long b = w0 + k;
        sd[k] = (b >= 0 && b <= n) ? D[b] : (signed char)-1;
    }
    __syncthreads();
    long long i = i0 + threadIdx.x;
    if (i >= n) return;
    int dl = min(level_for_limit(sd, w0, i, n, n_leaf), PETAR_MAXLEVEL);
    int gl_raw = level_for_limit(sd, w0, i, n, n_group);
    int gl = min(min(gl_raw, PETAR_MAXLEVEL), dl);
    depth[i] = (signed char)dl;
    glevel[i] = (signed char)gl;
    int flag;
    if (gl_raw > PETAR_MAXLEVEL) {
        // over-full level-21 cell: cut into consecutive chunks of n_group from the cell's first particle
        unsigned long long kk = key[i];
        long long lo = 0, hi = i;                 // first index with key == kk
        while (lo < hi) { long long mid = (lo + hi) >> 1; if (key[mid] < kk) lo = mid + 1; else hi = mid; }
        flag = ((i - lo) % n_group) == 0;
    } else {
        flag = (int)sd[i - w0] < gl;
    }
    gflag[i] = flag;
}

// ---- node ranking: id(i, l) = level_off[l] + (#level-l nodes starting before boundary i) ----------
#define RANK_THREADS 1024
__global__ void __launch_bounds__(RANK_THREADS) k_rank_count(const signed char* __restrict__ D, const signed char* __restrict__ depth,
                                                             long long n, int* __restrict__ tile_cnt, int ntile) {
    __shared__ int cnt[PETAR_NLEVELS];
    if (threadIdx.x < PETAR_NLEVELS) cnt[threadIdx.x] = 0;
    __syncthreads();
    long long i = (long long)blockIdx.x * RANK_THREADS + threadIdx.x;
    if (i < n) {
        int lo = D[i] + 1, hi = depth[i];
        for (int l = lo; l <= hi; ++l) atomicAdd(&cnt[l], 1);
    }
    __syncthreads();
    if (threadIdx.x < PETAR_NLEVELS) tile_cnt[threadIdx.x * ntile + blockIdx.x] = cnt[threadIdx.x];
}

// One CTA per tree level: exclusive scan of the level's per-tile node counts, in place (warp shuffles, two barriers per
// 1024 tiles).  Each CTA leaves its level's total in level_off[l]; the last CTA to finish turns the totals into the level
// offsets, sets the node count and checks the capacity.  (A single CTA doing the 22 levels one after the other took 0.36 ms
// at N = 10^7.)
__global__ void __launch_bounds__(1024) k_rank_scan(int* __restrict__ tile_cnt, int ntile, DevHeader* __restrict__ h, int node_cap) {
    __shared__ int wsum[32];
    __shared__ int carry_s, last_s;
    const int t = threadIdx.x, lane = t & 31, wp = t >> 5, l = blockIdx.x;
    int* row = tile_cnt + (size_t)l * ntile;
    if (t == 0) carry_s = 0;
    __syncthreads();
    for (int b0 = 0; b0 < ntile; b0 += 1024) {
        const int b = b0 + t;
        const int v = (b < ntile) ? row[b] : 0;
        int incl = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int a = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += a; }
        if (lane == 31) wsum[wp] = incl;
        __syncthreads();
        if (wp == 0) {
            const int sv = wsum[lane];
            int si = sv;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const int a = __shfl_up_sync(0xffffffffu, si, o); if (lane >= o) si += a; }
            wsum[lane] = si - sv;                       // tiles of the warps before this one
        }
        __syncthreads();
        const int excl = carry_s + wsum[wp] + incl - v;
        if (b < ntile) row[b] = excl;
        __syncthreads();                                // carry_s and wsum read by everybody
        if (t == 1023) carry_s = excl + v;
        __syncthreads();
    }
    if (t == 0) {
        ((volatile int*)h->level_off)[l] = carry_s;     // this level's total, for now
        __threadfence();
        last_s = atomicAdd(&h->rank_done, 1) == (int)gridDim.x - 1;
    }
    __syncthreads();
    if (last_s && t == 0) {
        __threadfence();
        int run = 0;
        for (int k = 0; k < PETAR_NLEVELS; ++k) { const int c = ((volatile int*)h->level_off)[k]; h->level_off[k] = run; run += c; }
        h->level_off[PETAR_NLEVELS] = run; h->level_off[PETAR_NLEVELS + 1] = run;
        h->n_nodes = run;
        if (run > node_cap) { atomicOr(&h->status, PETAR_ST_NODE_CAP); }
        h->rank_done = 0;
    }
}

__global__ void __launch_bounds__(RANK_THREADS) k_nodes_write(const unsigned long long* __restrict__ key, const signed char* __restrict__ D,
                                                              const signed char* __restrict__ depth, long long n,
                                                              const int* __restrict__ tile_off, int ntile, const DevHeader* __restrict__ h,
                                                              NodeInt* __restrict__ nint, int node_cap) {
    __shared__ unsigned s_bal[RANK_THREADS / 32][PETAR_NLEVELS];
    __shared__ int s_woff[RANK_THREADS / 32][PETAR_NLEVELS];
    const int t = threadIdx.x, lane = t & 31, w = t >> 5;
    const long long i = (long long)blockIdx.x * RANK_THREADS + t;
    int lo = 1, hi = 0;
    if (i < n) { lo = D[i] + 1; hi = depth[i]; }
#pragma unroll
    for (int l = 0; l < PETAR_NLEVELS; ++l) {
        unsigned bal = __ballot_sync(0xffffffffu, l >= lo && l <= hi);
        if (lane == 0) s_bal[w][l] = bal;
    }
    __syncthreads();
    if (t < PETAR_NLEVELS) {
        int run = h->level_off[t] + tile_off[(size_t)t * ntile + blockIdx.x];
        for (int ww = 0; ww < RANK_THREADS / 32; ++ww) { s_woff[ww][t] = run; run += __popc(s_bal[ww][t]); }
    }
    __syncthreads();
    if (h->n_nodes > node_cap) return;            // capacity exceeded: status already set
    if (i >= n || lo > hi) return;
    const unsigned lt = (1u << lane) - 1u;
    const unsigned long long ki = key[i];
    for (int l = lo; l <= hi; ++l) {
        int id = s_woff[w][l] + __popc(s_bal[w][l] & lt);
        int child = (l < hi) ? (s_woff[w][l + 1] + __popc(s_bal[w][l + 1] & lt)) : -1;
        // end of the cell: first j > i whose level-l prefix differs (galloping + binary search)
        long long end;
        if (l == 0) end = n;
        else {
            const int shift = 3 * (PETAR_MAXLEVEL - l);
            const unsigned long long pref = ki >> shift;
            long long a = i, step = 1;
            while (a + step < n && (key[a + step] >> shift) == pref) { a += step; step <<= 1; }
            long long b = min(n, a + step);        // key[a] matches, key[b] differs or b == n
            while (b - a > 1) { long long mid = (a + b) >> 1; if ((key[mid] >> shift) == pref) a = mid; else b = mid; }
            end = b;
        }
        NodeInt r;
        r.begin = (int)i; r.end = (int)end; r.first_child = child;
        r.meta = l | ((l == hi) ? (1 << 16) : 0) | ((l > lo) ? (1 << 17) : 0);
        nint[id] = r;
    }
}

// ------------------------------------------------------------------------------------------------
// S5: bottom-up moments, one level per grid-wide phase (cooperative launch).  Summation order is
// rule O5: leaf = members in sorted order with S = fma(m, x, S); internal = children ascending.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_moments(const DevHeader* __restrict__ h, NodeInt* __restrict__ nint, NodeMac* __restrict__ nmac,
                                                 NodeMom* __restrict__ nmom, NodeSp* __restrict__ nsp, NodeW* __restrict__ nw,
                                                 const unsigned long long* __restrict__ key,
                                                 const double* __restrict__ xs, const double* __restrict__ ys, const double* __restrict__ zs,
                                                 const double* __restrict__ ms, const double* __restrict__ rss, int node_cap, int multipole) {
    cg::grid_group grid = cg::this_grid();
    if (h->n_nodes > node_cap) return;            // uniform across the grid
    const long long gsz = (long long)gridDim.x * blockDim.x;
    const long long gtid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const double cx = h->c[0], cy = h->c[1], cz = h->c[2];
    for (int l = PETAR_MAXLEVEL; l >= 0; --l) {
        const int n0 = h->level_off[l], n1 = h->level_off[l + 1], n2 = h->level_off[l + 2];
        if (n0 == n1) continue;                    // empty level (uniform across the grid): no phase, no grid barrier
        for (long long id = n0 + gtid; id < n1; id += gsz) {
            NodeInt r = nint[id];
            double M = 0, S0 = 0, S1 = 0, S2 = 0, rmax = 0;
            double lo0 = INFINITY, lo1 = INFINITY, lo2 = INFINITY, hi0 = -INFINITY, hi1 = -INFINITY, hi2 = -INFINITY;
            double Q[6] = {0, 0, 0, 0, 0, 0};
            double com0, com1, com2;
            const bool leaf = (r.meta >> 16) & 1;
            int nchild = 0;
            if (leaf) {
                for (int p = r.begin; p < r.end; ++p) {
                    double m = ms[p], x = xs[p], y = ys[p], z = zs[p];
                    M = M + m;
                    S0 = fma(m, x, S0); S1 = fma(m, y, S1); S2 = fma(m, z, S2);
                    lo0 = fmin(lo0, x); lo1 = fmin(lo1, y); lo2 = fmin(lo2, z);
                    hi0 = fmax(hi0, x); hi1 = fmax(hi1, y); hi2 = fmax(hi2, z);
                    rmax = fmax(rmax, rss[p]);
                }
            } else {
                int c = r.first_child;
                do {
                    NodeMom cm = nmom[c];
                    NodeMac cc = nmac[c];
                    M = M + cm.M; S0 = S0 + cm.S[0]; S1 = S1 + cm.S[1]; S2 = S2 + cm.S[2];
                    lo0 = fmin(lo0, cc.lo[0]); lo1 = fmin(lo1, cc.lo[1]); lo2 = fmin(lo2, cc.lo[2]);
                    hi0 = fmax(hi0, cc.hi[0]); hi1 = fmax(hi1, cc.hi[1]); hi2 = fmax(hi2, cc.hi[2]);
                    rmax = fmax(rmax, cc.rmax);
                    ++c; ++nchild;
                } while (nchild < 8 && c < n2 && !((nint[c].meta >> 17) & 1));
            }
            if (M != 0.0) { com0 = S0 / M; com1 = S1 / M; com2 = S2 / M; }
            else {
                // massless cell: centre of its cube
                unsigned long long pref = l ? (key[r.begin] >> (3 * (PETAR_MAXLEVEL - l))) << (3 * (PETAR_MAXLEVEL - l)) : 0ull;
                double edge = ldexp(2.0 * h->h, -l);
                int sh = PETAR_MAXLEVEL - l;
                double q0 = (double)(compact21(pref >> 2) >> sh), q1 = (double)(compact21(pref >> 1) >> sh), q2 = (double)(compact21(pref) >> sh);
                com0 = h->o[0] + (q0 + 0.5) * edge; com1 = h->o[1] + (q1 + 0.5) * edge; com2 = h->o[2] + (q2 + 0.5) * edge;
            }
            // quadrupole about com (Eq. 30): any summation order is allowed (tolerance-compared only)
            if (leaf) {
                for (int p = r.begin; p < r.end; ++p) {
                    double m = ms[p], dx = xs[p] - com0, dy = ys[p] - com1, dz = zs[p] - com2;
                    Q[0] += m * dx * dx; Q[1] += m * dy * dy; Q[2] += m * dz * dz;
                    Q[3] += m * dx * dy; Q[4] += m * dx * dz; Q[5] += m * dy * dz;
                }
            } else {
                for (int k = 0; k < nchild; ++k) {        // parallel-axis rule
                    int c = r.first_child + k;
                    NodeMom cm = nmom[c];
                    NodeMac cc = nmac[c];
                    double dx = cc.com[0] - com0, dy = cc.com[1] - com1, dz = cc.com[2] - com2;
                    Q[0] += cm.Q[0] + cm.M * dx * dx; Q[1] += cm.Q[1] + cm.M * dy * dy; Q[2] += cm.Q[2] + cm.M * dz * dz;
                    Q[3] += cm.Q[3] + cm.M * dx * dy; Q[4] += cm.Q[4] + cm.M * dx * dz; Q[5] += cm.Q[5] + cm.M * dy * dz;
                }
                r.meta |= (nchild << 8);
                nint[id].meta = r.meta;
            }
            NodeMac mac;
            mac.lo[0] = lo0; mac.lo[1] = lo1; mac.lo[2] = lo2; mac.hi[0] = hi0; mac.hi[1] = hi1; mac.hi[2] = hi2;
            mac.com[0] = com0; mac.com[1] = com1; mac.com[2] = com2; mac.rmax = rmax;
            nmac[id] = mac;
            NodeMom mom;
            mom.M = M; mom.S[0] = S0; mom.S[1] = S1; mom.S[2] = S2;
            for (int k = 0; k < 6; ++k) mom.Q[k] = Q[k];
            nmom[id] = mom;
            // fp32 super-particle record: float-float position relative to the root centre, traceless A'
            double dx = com0 - cx, dy = com1 - cy, dz = com2 - cz;
            float xh = (float)dx, yh = (float)dy, zh = (float)dz;
            float xl = (float)(dx - (double)xh), yl = (float)(dy - (double)yh), zl = (float)(dz - (double)zh);
            double tr = Q[0] + Q[1] + Q[2];
            NodeSp sp;
            sp.q0 = make_float4(xh, yh, zh, (float)M);
            if (multipole >= 2) {
                // B = -2 A' with A' = 1.5 Q - 0.5 tr(Q) I  (the force kernel works with B, see force.cu)
                sp.q1 = make_float4(xl, yl, zl, (float)(-2.0 * (1.5 * Q[0] - 0.5 * tr)));
                sp.q2 = make_float4((float)(-2.0 * (1.5 * Q[1] - 0.5 * tr)), (float)(-3.0 * Q[3]), (float)(-3.0 * Q[4]), (float)(-3.0 * Q[5]));
            } else {
                sp.q1 = make_float4(xl, yl, zl, 0.f);
                sp.q2 = make_float4(0.f, 0.f, 0.f, 0.f);
            }
            nsp[id] = sp;
            // fp32 walk record: coordinates relative to the root centre, error bound eps
            {
                NodeW wr;
                const float l0 = (float)(lo0 - cx), l1 = (float)(lo1 - cy), l2 = (float)(lo2 - cz);
                const float h0 = (float)(hi0 - cx), h1 = (float)(hi1 - cy), h2 = (float)(hi2 - cz);
                // largest |coordinate| of anything the walk's fp32 tests read from this record: the tight box and the centre of
                // mass (for a massless cell, or with negative masses, the latter can lie outside the box)
                const float amax = fmaxf(fmaxf(fmaxf(fmaxf(fabsf(l0), fabsf(h0)), fmaxf(fabsf(l1), fabsf(h1))), fmaxf(fabsf(l2), fabsf(h2))),
                                         fmaxf(fmaxf(fabsf(xh), fabsf(yh)), fabsf(zh)));
                wr.a = make_float4(l0, l1, l2, h0);
                wr.b = make_float4(h1, h2, xh, yh);
                wr.c = make_float4(zh, (float)rmax, amax * 4.8e-7f, 0.f);
                wr.d = make_int4(r.begin, r.end, r.first_child, r.meta);
                nw[id] = wr;
            }
        }
        grid.sync();
    }
}

// ------------------------------------------------------------------------------------------------
// S6: i-groups from the scanned start flags
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_groups_begin(const int* __restrict__ gflag, const int* __restrict__ gscan, long long n,
                                                      GroupRec* __restrict__ grp, DevHeader* __restrict__ h) {
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i == 0) h->n_groups = gscan[n];
    if (i >= n) return;
    if (gflag[i]) grp[gscan[i]].begin = (int)i;
}

// one warp per group: end, tight box, rmax; list heads reset
__global__ void __launch_bounds__(256) k_groups_finish(GroupRec* __restrict__ grp, const DevHeader* __restrict__ h, long long n,
                                                       const double* __restrict__ xs, const double* __restrict__ ys, const double* __restrict__ zs,
                                                       const double* __restrict__ rss) {
    const int lane = threadIdx.x & 31;
    const int ng = h->n_groups;
    for (long long g = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5; g < ng; g += ((long long)gridDim.x * blockDim.x) >> 5) {
        int b = grp[g].begin;
        int e = (g + 1 < ng) ? grp[g + 1].begin : (int)n;
        double lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY}, rmax = 0;
        for (int p = b + lane; p < e; p += 32) {
            double v[3] = {xs[p], ys[p], zs[p]};
#pragma unroll
            for (int k = 0; k < 3; ++k) { lo[k] = fmin(lo[k], v[k]); hi[k] = fmax(hi[k], v[k]); }
            rmax = fmax(rmax, rss[p]);
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) {
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                lo[k] = fmin(lo[k], __shfl_xor_sync(0xffffffffu, lo[k], o));
                hi[k] = fmax(hi[k], __shfl_xor_sync(0xffffffffu, hi[k], o));
            }
            rmax = fmax(rmax, __shfl_xor_sync(0xffffffffu, rmax, o));
        }
        __syncwarp();
        if (lane == 0) {          // (begin is left alone: the neighbouring warp reads it)
            GroupRec* r = &grp[g];
            r->end = e; r->head_sp = r->head_epn = r->head_epf = -1;
            r->n_sp = r->n_epn = r->n_epf = 0; r->n_ep_part = r->n_epn_part = 0; r->head_spp = -1; r->n_spp = 0;
            for (int k = 0; k < 3; ++k) { r->lo[k] = lo[k]; r->hi[k] = hi[k]; }
            r->rmax = rmax; for (int l = 0; l < PETAR_NSUP; ++l) r->sid[l] = 0;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// device-wide exclusive scans (reduce -> scan of partials -> scan + add), 4096 elements per CTA
// ------------------------------------------------------------------------------------------------
#define SCAN_THREADS 1024
#define SCAN_ITEMS 4
template <typename T>
__device__ __forceinline__ T block_excl_scan(T v, T* total_out, T* sbuf /* 32 */) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    T incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { T a = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += a; }
    if (lane == 31) sbuf[w] = incl;
    __syncthreads();
    if (w == 0) {
        T x = (lane < (int)(blockDim.x >> 5)) ? sbuf[lane] : (T)0;
        T xi = x;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { T a = __shfl_up_sync(0xffffffffu, xi, o); if (lane >= o) xi += a; }
        sbuf[lane] = xi - x;
        if (lane == 31) *total_out = xi;
    }
    __syncthreads();
    T r = sbuf[w] + incl - v;
    __syncthreads();
    return r;
}

template <typename TO>
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_reduce(const int* __restrict__ in, long long n, TO* __restrict__ part) {
    __shared__ TO sbuf[32];
    __shared__ TO tot;
    long long base = (long long)blockIdx.x * SCAN_THREADS * SCAN_ITEMS + (long long)threadIdx.x * SCAN_ITEMS;
    TO s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) if (base + k < n) s += (TO)in[base + k];
    (void)block_excl_scan<TO>(s, &tot, sbuf);
    if (threadIdx.x == 0) part[blockIdx.x] = tot;
}
template <typename TO>
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_partials(TO* __restrict__ part, int nblk) {
    __shared__ TO sbuf[32];
    __shared__ TO tot;
    __shared__ TO carry_s;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int b0 = 0; b0 < nblk; b0 += SCAN_THREADS) {
        int b = b0 + threadIdx.x;
        TO v = (b < nblk) ? part[b] : (TO)0;
        TO ex = block_excl_scan<TO>(v, &tot, sbuf);
        TO carry = carry_s;
        if (b < nblk) part[b] = carry + ex;
        __syncthreads();
        if (threadIdx.x == 0) carry_s = carry + tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) part[nblk] = carry_s;
}
template <typename TO>
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_final(const int* __restrict__ in, long long n, const TO* __restrict__ part,
                                                             int nblk, TO* __restrict__ out) {
    __shared__ TO sbuf[32];
    __shared__ TO tot;
    long long base = (long long)blockIdx.x * SCAN_THREADS * SCAN_ITEMS + (long long)threadIdx.x * SCAN_ITEMS;
    int v[SCAN_ITEMS];
    TO s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) { v[k] = (base + k < n) ? in[base + k] : 0; s += (TO)v[k]; }
    TO ex = block_excl_scan<TO>(s, &tot, sbuf) + part[blockIdx.x];
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) { if (base + k < n) out[base + k] = ex; ex += (TO)v[k]; }
    if (blockIdx.x == 0 && threadIdx.x == 0) out[n] = part[nblk];
}

template <typename TO>
static cudaError_t scan_impl(const int* in, TO* out, long long n, TO* tmp, cudaStream_t s) {
    int nblk = cdiv(n, SCAN_THREADS * SCAN_ITEMS);
    if (nblk < 1) nblk = 1;
    k_scan_reduce<TO><<<nblk, SCAN_THREADS, 0, s>>>(in, n, tmp);
    KCHECK(s, "k_scan_reduce");
    k_scan_partials<TO><<<1, SCAN_THREADS, 0, s>>>(tmp, nblk);
    KCHECK(s, "k_scan_partials");
    k_scan_final<TO><<<nblk, SCAN_THREADS, 0, s>>>(in, n, tmp, nblk, out);
    KCHECK(s, "k_scan_final");
    petar_count_launch(3);
    return cudaGetLastError();
}
cudaError_t launch_scan_i32(const int* in, int* out, int n, int* tmp, cudaStream_t s) { return scan_impl<int>(in, out, n, tmp, s); }
cudaError_t launch_scan_i32_to_i64(const int* in, long long* out, long long n, long long* tmp, cudaStream_t s) {
    return scan_impl<long long>(in, out, n, tmp, s);
}

// ------------------------------------------------------------------------------------------------
// host-side launch sequences
// ------------------------------------------------------------------------------------------------
int radix_sort_blocks(long long n) { return cdiv(n, SORT_TILE); }

cudaError_t launch_radix_sort(unsigned long long* key, unsigned long long* key_alt, unsigned* idx, unsigned* idx_alt,
                              unsigned* hist, unsigned* blk, long long n, int npass, cudaStream_t s) {
    const int nblk = cdiv(n, SORT_TILE);
    cudaError_t e = cudaMemsetAsync(hist, 0, (size_t)npass * 256 * sizeof(unsigned), s);
    if (e != cudaSuccess) return e;
    unsigned long long *kin = key, *kout = key_alt;
    unsigned *vin = idx, *vout = idx_alt;
    for (int pass = 0; pass < npass; ++pass) {
        int shift = 8 * pass;
        k_sort_count<<<nblk, SORT_THREADS, 0, s>>>(kin, n, shift, blk, nblk, hist + 256 * pass);
        KCHECK(s, "k_sort_count");
        k_sort_scan<<<256, 256, 0, s>>>(blk, nblk, hist + 256 * pass);
        KCHECK(s, "k_sort_scan");
        k_sort_scatter<<<nblk, SORT_THREADS, 0, s>>>(kin, vin, kout, vout, blk, nblk, n, shift);
        KCHECK(s, "k_sort_scatter");
        unsigned long long* tk = kin; kin = kout; kout = tk;
        unsigned* tv = vin; vin = vout; vout = tv;
    }
    petar_count_launch(3 * npass);
    return cudaGetLastError();
}

// Eq. 24, rule O10a: r_nb = r_out + (C_r sqrt(v2)) dt, v2 = fma(vz,vz, fma(vy,vy, vx*vx))
__global__ void __launch_bounds__(256) k_search_radii(const double* __restrict__ vx, const double* __restrict__ vy, const double* __restrict__ vz,
                                                      const double* __restrict__ rout, double Cr, double dt, long long n, double* __restrict__ out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double v2 = fma(vz[i], vz[i], fma(vy[i], vy[i], vx[i] * vx[i]));
    out[i] = rout[i] + (Cr * sqrt(v2)) * dt;
}
cudaError_t launch_search_radii(const double* vx, const double* vy, const double* vz, const double* r_out, double Cr, double dt,
                                long long n, double* out, cudaStream_t s) {
    if (n > 0) k_search_radii<<<cdiv(n, 256), 256, 0, s>>>(vx, vy, vz, r_out, Cr, dt, n, out);
    KCHECK(s, "k_search_radii");
    petar_count_launch(1);
    return cudaGetLastError();
}

cudaError_t launch_keys_sort_gather(petar_tree* t, cudaStream_t s) {
    Workspace& w = t->w;
    const long long n = t->N;
    stage_begin(t, PETAR_STAGE_BBOX_KEYS, s);
    k_reset_header<<<1, 32, 0, s>>>(w.hdr);
    KCHECK(s, "k_reset_header");
    int g = min(cdiv(n, 256), t->sm_count * 8);
    k_bbox<<<g, 256, 0, s>>>(t->x, t->y, t->z, n, w.hdr);
    KCHECK(s, "k_bbox");
    k_root<<<1, 32, 0, s>>>(w.hdr);
    KCHECK(s, "k_root");
    k_keys<<<cdiv(n, 512), 256, 0, s>>>(t->x, t->y, t->z, t->m, t->r_out, t->r_search, n, w.hdr, w.key, w.idx, w.rec);
    KCHECK(s, "k_keys");
    petar_count_launch(4);
    stage_end(t, PETAR_STAGE_BBOX_KEYS, s);

    stage_begin(t, PETAR_STAGE_SORT, s);
    {
        cudaError_t e = launch_radix_sort(w.key, w.key_alt, w.idx, w.idx_alt, w.sort_hist, w.sort_blk, n, 8, s);
        if (e != cudaSuccess) return e;
    }
    // 8 passes: the sorted data is back in (key, idx)
    stage_end(t, PETAR_STAGE_SORT, s);

    stage_begin(t, PETAR_STAGE_GATHER, s);
    k_gather<<<cdiv(n, 256), 256, 0, s>>>(w.idx, n, w.hdr, w.rec, t->r_search != nullptr,
                                          w.xs, w.ys, w.zs, w.ms, w.routs, t->r_search ? w.rss : nullptr, w.pa, w.pb);
    KCHECK(s, "k_gather");
    petar_count_launch(1);
    stage_end(t, PETAR_STAGE_GATHER, s);
    return cudaGetLastError();
}

cudaError_t launch_tree(petar_tree* t, cudaStream_t s) {
    Workspace& w = t->w;
    const long long n = t->N;
    const int ntile = cdiv(n, RANK_THREADS);
    stage_begin(t, PETAR_STAGE_TREE, s);
    k_diverge<<<cdiv(n + 1, 256), 256, 0, s>>>(w.key, n, w.D);
    KCHECK(s, "k_diverge");
    size_t sh = DEPTH_THREADS + 2 * t->p.n_group_limit + 1;
    k_depth<<<cdiv(n, DEPTH_THREADS), DEPTH_THREADS, sh, s>>>(w.key, w.D, n, t->p.n_leaf_limit, t->p.n_group_limit, w.depth, w.glevel, w.gflag);
    KCHECK(s, "k_depth");
    k_rank_count<<<ntile, RANK_THREADS, 0, s>>>(w.D, w.depth, n, w.tile_cnt, ntile);
    KCHECK(s, "k_rank_count");
    k_rank_scan<<<PETAR_NLEVELS, 1024, 0, s>>>(w.tile_cnt, ntile, w.hdr, w.node_cap);
    KCHECK(s, "k_rank_scan");
    k_nodes_write<<<ntile, RANK_THREADS, 0, s>>>(w.key, w.D, w.depth, n, w.tile_cnt, ntile, w.hdr, w.nint, w.node_cap);
    KCHECK(s, "k_nodes_write");
    petar_count_launch(5);
    stage_end(t, PETAR_STAGE_TREE, s);

    stage_begin(t, PETAR_STAGE_MOMENTS, s);
    {
        int per_sm = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_moments, 256, 0);
        if (e != cudaSuccess) return e;
        if (per_sm < 1) per_sm = 1;
        if (per_sm > 4) per_sm = 4;
        int grid = t->sm_count * per_sm;
        const DevHeader* hdr = w.hdr;
        const double* rss = t->r_search ? w.rss : w.routs;
        int cap = w.node_cap, mult = t->p.multipole;
        void* args[] = {(void*)&hdr, (void*)&w.nint, (void*)&w.nmac, (void*)&w.nmom, (void*)&w.nsp, (void*)&w.nw, (void*)&w.key,
                        (void*)&w.xs, (void*)&w.ys, (void*)&w.zs, (void*)&w.ms, (void*)&rss, (void*)&cap, (void*)&mult};
        e = cudaLaunchCooperativeKernel((void*)k_moments, dim3(grid), dim3(256), args, 0, s);
        if (e != cudaSuccess) return e;
        KCHECK(s, "k_moments");
        petar_count_launch(1);
    }
    stage_end(t, PETAR_STAGE_MOMENTS, s);

    stage_begin(t, PETAR_STAGE_GROUPS, s);
    cudaError_t e = launch_scan_i32(w.gflag, w.gflag + (n + 1), (int)n, w.scan_tmp, s);
    if (e != cudaSuccess) return e;
    k_groups_begin<<<cdiv(n, 256), 256, 0, s>>>(w.gflag, w.gflag + (n + 1), n, w.grp, w.hdr);
    KCHECK(s, "k_groups_begin");
    k_groups_finish<<<min(cdiv(n, 8), t->sm_count * 16), 256, 0, s>>>(w.grp, w.hdr, n, w.xs, w.ys, w.zs, t->r_search ? w.rss : w.routs);
    KCHECK(s, "k_groups_finish");
    petar_count_launch(2);
    stage_end(t, PETAR_STAGE_GROUPS, s);
    return cudaGetLastError();
}

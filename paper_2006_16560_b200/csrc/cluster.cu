// cluster.cu -- clustering of the neighbour graph: "any member in one cluster have all
// its neighbours inside the same cluster", i.e. the clusters are the connected components of the
// (symmetric) neighbour list.  Lock-free union-find on the device: the larger root is always hooked
// under the smaller one, so the final root of a component is its smallest member whatever the order in
// which the edges are processed -- the labels are deterministic.  No host synchronisation.
// Member lists: stable radix sort of (label, particle index), cluster starts by a flag scan.
#include "internal.cuh"

// multiprocessors of the CURRENT device (asked on every call: a process may drive several GPUs, and the query is a host-side lookup)
static int sm_count() {
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
    return n;
}

__device__ __forceinline__ int cc_find(int* __restrict__ parent, int a) {
    int p = ((volatile int*)parent)[a];
    while (p != a) {
        const int gp = ((volatile int*)parent)[p];
        if (gp != p) atomicMin(&parent[a], gp);         // path halving (parents only ever decrease)
        a = p; p = gp;
    }
    return a;
}

__global__ void __launch_bounds__(256) k_cc_init(int* __restrict__ parent, long long n, long long* __restrict__ n_clusters) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0 && n_clusters) *n_clusters = 0;
    if (i < n) parent[i] = (int)i;
}

// one thread per edge entry: row lookup by binary search in the offsets
__global__ void __launch_bounds__(256) k_cc_union(const long long* __restrict__ offsets, const int* __restrict__ indices, long long n,
                                                  int* __restrict__ parent) {
    const long long total = offsets[n];
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
        long long lo = 0, hi = n;                      // largest i with offsets[i] <= e
        while (hi - lo > 1) { const long long mid = (lo + hi) >> 1; if (offsets[mid] <= e) lo = mid; else hi = mid; }
        int a = (int)lo, b = indices[e];
        if (b < 0 || b >= n || b == a) continue;
        for (;;) {
            a = cc_find(parent, a); b = cc_find(parent, b);
            if (a == b) break;
            if (a < b) { const int t = a; a = b; b = t; }      // a > b: hook root a under b
            const int old = atomicCAS(&parent[a], a, b);
            if (old == a) break;
            a = old;                                    // a was no root any more: retry from its new parent
        }
    }
}

__global__ void __launch_bounds__(256) k_cc_flatten(int* __restrict__ parent, long long n, long long* __restrict__ n_clusters) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int root = 0;
    bool is_root = false;
    if (i < n) {
        root = (int)i;
        int p = ((volatile int*)parent)[root];
        while (p != root) { root = p; p = ((volatile int*)parent)[root]; }
        is_root = root == (int)i;
    }
    // roots never change in this kernel (only non-roots are rewritten), so the walks above stay valid
    if (i < n && !is_root) parent[i] = root;
    const unsigned m = __ballot_sync(0xffffffffu, is_root);
    if (n_clusters && (threadIdx.x & 31) == 0 && m) atomicAdd((unsigned long long*)n_clusters, (unsigned long long)__popc(m));
}

__global__ void __launch_bounds__(256) k_cc_keys(const int* __restrict__ label, long long n, unsigned long long* __restrict__ key, unsigned* __restrict__ idx) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { key[i] = (unsigned long long)(unsigned)label[i]; idx[i] = (unsigned)i; }
}
__global__ void __launch_bounds__(256) k_cc_flags(const unsigned long long* __restrict__ key, long long n, int* __restrict__ flag) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) flag[i] = (i == 0 || key[i] != key[i - 1]) ? 1 : 0;
}
// rank[i] = clusters that start before sorted position i; a start at i writes cluster_offsets[rank[i]] = i
__global__ void __launch_bounds__(256) k_cc_offsets(const int* __restrict__ flag, const int* __restrict__ rank, const unsigned* __restrict__ idx,
                                                    long long n, long long* __restrict__ cluster_offsets, int* __restrict__ members) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        if (members) members[i] = (int)idx[i];
        if (flag[i]) cluster_offsets[rank[i]] = i;
    }
    if (i == n) cluster_offsets[rank[n]] = n;           // rank[n] = number of clusters
}

static inline size_t al256(size_t v) { return (v + 255) / 256 * 256; }
size_t clusters_workspace_bytes(long long n) {
    const size_t N = (size_t)(n > 0 ? n : 0);
    const int nblk = radix_sort_blocks(n) + 1;
    return al256(N * 8) * 2 + al256(N * 4) * 2 + al256(4 * 256 * 4) + al256((size_t)256 * nblk * 4) + al256((N + 1) * 4) * 2 + al256((N / 4096 + 8) * 8) + 256;
}

cudaError_t launch_clusters(const long long* offsets, const int* indices, long long n, int* label, long long* n_clusters_dev,
                            long long* cluster_offsets, int* members, void* workspace, cudaStream_t s) {
    if (n <= 0) return cudaSuccess;
    const int nb = cdiv(n, 256);
    k_cc_init<<<nb, 256, 0, s>>>(label, n, n_clusters_dev);
    KCHECK(s, "k_cc_init");
    k_cc_union<<<sm_count() * 16, 256, 0, s>>>(offsets, indices, n, label);
    KCHECK(s, "k_cc_union");
    k_cc_flatten<<<nb, 256, 0, s>>>(label, n, n_clusters_dev);
    KCHECK(s, "k_cc_flatten");
    petar_count_launch(3);
    if (!cluster_offsets) return cudaGetLastError();
    // member lists
    char* base = (char*)workspace;
    size_t off = 0;
    auto take = [&](size_t bytes) { char* r = base + off; off += al256(bytes); return r; };
    const size_t N = (size_t)n;
    const int nblk = radix_sort_blocks(n) + 1;
    unsigned long long* key = (unsigned long long*)take(N * 8); unsigned long long* key_alt = (unsigned long long*)take(N * 8);
    unsigned* idx = (unsigned*)take(N * 4); unsigned* idx_alt = (unsigned*)take(N * 4);
    unsigned* hist = (unsigned*)take(4 * 256 * 4); unsigned* blk = (unsigned*)take((size_t)256 * nblk * 4);
    int* flag = (int*)take((N + 1) * 4); int* rank = (int*)take((N + 1) * 4);
    int* tmp = (int*)take((N / 4096 + 8) * 8);
    k_cc_keys<<<nb, 256, 0, s>>>(label, n, key, idx);
    KCHECK(s, "k_cc_keys");
    cudaError_t e = launch_radix_sort(key, key_alt, idx, idx_alt, hist, blk, n, 4, s);     // labels are < 2^31: 4 passes
    if (e != cudaSuccess) return e;
    k_cc_flags<<<nb, 256, 0, s>>>(key, n, flag);
    KCHECK(s, "k_cc_flags");
    e = launch_scan_i32(flag, rank, (int)n, tmp, s);
    if (e != cudaSuccess) return e;
    k_cc_offsets<<<cdiv(n + 1, 256), 256, 0, s>>>(flag, rank, idx, n, cluster_offsets, members);
    KCHECK(s, "k_cc_offsets");
    petar_count_launch(3);
    return cudaGetLastError();
}

// short.cu -- SURVEY.md 8(f) rank 4: the short-range part H_S of Eq. 11 over the
// neighbour rows: acceleration, its first time derivative (the Hermite integrator's force evaluation,
// PAPER.md:300, Eq. 40 :639) and potential, with the changeover functions K (Eq. 17), W (Eq. 15) and
// K' = -280 Lambda (x+q) x^3 (1-x)^3 (from Eq. 18).  All fp64.
//
// Rows are short (the binary companion, rarely a few more) with a few very long ones (a massive
// particle): rows of up to SHORT_ROW entries are summed by one thread in list order; longer rows are
// queued and summed by one warp each (lanes take entries lane, lane+32, ..., then a fixed-order
// shuffle reduction), so every result is deterministic.  HBM-bound: the inputs are first packed into one
// 64-byte record per particle (64 B read + 64 B written), then 64 B read + 56 B written per particle and one
// 64-byte record gathered per list entry.
#include "internal.cuh"
#include <mutex>

// multiprocessors of the CURRENT device (asked on every call: a process may drive several GPUs, and the query is a host-side lookup)
static int sm_count() {
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
    return n;
}

#define SHORT_ROW 32

// packed copy of the inputs: one 64-byte record per particle, so a gathered neighbour costs two sectors, not eight
struct __align__(16) ShortRec { double x, y, z, vx, vy, vz, m, rout; };

struct ShortArgs {
    const double *x, *y, *z, *vx, *vy, *vz, *m, *rout;
    const ShortRec* rec;
    const long long* offsets; const int* indices;
    double *ax, *ay, *az, *jx, *jy, *jz, *pot;
    double G, rho, lam, q;
    long long n;
};

struct Sum7 { double a0, a1, a2, j0, j1, j2, p; };

__device__ __forceinline__ void short_pair(const ShortArgs& A, const double xi, const double yi, const double zi, const double vxi,
                                           const double vyi, const double vzi, const double ri, const int j, Sum7& s) {
    const double2* rp = reinterpret_cast<const double2*>(&A.rec[j]);
    const double2 q0 = rp[0], q1 = rp[1], q2 = rp[2], q3 = rp[3];         // (x, y) (z, vx) (vy, vz) (m, rout)
    const double dx = xi - q0.x, dy = yi - q0.y, dz = zi - q1.x;
    const double wx = vxi - q1.y, wy = vyi - q2.x, wz = vzi - q2.y;
    const double r2 = dx * dx + dy * dy + dz * dz;
    const double r = sqrt(r2);
    const double R = fmax(ri, q3.y);
    if (r == 0.0 || r >= R) return;
    const double rin = A.rho * R;
    const double xx = (r - rin) / (R - rin);
    double K = 1.0, dK = 0.0, W;
    if (xx > 0.0) {
        const double xm = xx - 1.0, xm2 = xm * xm, x2 = xx * xx;
        K = (xm2 * xm2) * (1.0 + 4.0 * xx + 10.0 * x2 + 20.0 * x2 * xx + 35.0 * A.lam * x2 * x2);      // Eq. 17
        const double y = 1.0 - xx;
        dK = -280.0 * A.lam * (xx + A.q) * (x2 * xx) * (y * y * y);
        W = A.lam * (1.0 - 2.0 * xx) + A.lam * (x2 * x2 * xx) * (14.0 - 28.0 * xx + 20.0 * x2 - 5.0 * x2 * xx);   // Eq. 15: ... - 1 + f(x)
    } else {
        W = A.lam * (1.0 - 2.0 * xx);                                                                    // x <= 0, unclamped (reading P4)
    }
    const double mj = q3.x;
    const double dw = dx * wx + dy * wy + dz * wz;
    const double r3 = r2 * r;
    const double xdot = dw / (r * (R - rin));
    const double c0 = -A.G * mj * K / r3;
    const double c1 = -A.G * mj * (-3.0 * K * dw / (r3 * r2) + dK * xdot / r3);
    s.a0 += c0 * dx; s.a1 += c0 * dy; s.a2 += c0 * dz;
    s.j0 += c0 * wx + c1 * dx; s.j1 += c0 * wy + c1 * dy; s.j2 += c0 * wz + c1 * dz;
    s.p -= A.G * mj * W / r;
}

__device__ __forceinline__ void short_store(const ShortArgs& A, const long long i, const Sum7& s) {
    if (A.ax) A.ax[i] = s.a0; if (A.ay) A.ay[i] = s.a1; if (A.az) A.az[i] = s.a2;
    if (A.jx) A.jx[i] = s.j0; if (A.jy) A.jy[i] = s.j1; if (A.jz) A.jz[i] = s.j2;
    if (A.pot) A.pot[i] = s.p;
}

__global__ void __launch_bounds__(256) k_short_pack(const ShortArgs A, ShortRec* __restrict__ rec) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= A.n) return;
    ShortRec r = {A.x[i], A.y[i], A.z[i], A.vx[i], A.vy[i], A.vz[i], A.m[i], A.rout[i]};
    rec[i] = r;
}

// queue[0] = number of long rows, queue[1..] = their particle indices
__global__ void __launch_bounds__(256) k_short_rows(const ShortArgs A, int* __restrict__ queue) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= A.n) return;
    const long long b = A.offsets[i], e = A.offsets[i + 1];
    if (e - b > SHORT_ROW) { queue[1 + atomicAdd(&queue[0], 1)] = (int)i; return; }
    Sum7 s = {0, 0, 0, 0, 0, 0, 0};
    if (e > b) {
        const double xi = A.x[i], yi = A.y[i], zi = A.z[i], vxi = A.vx[i], vyi = A.vy[i], vzi = A.vz[i], ri = A.rout[i];
        for (long long k = b; k < e; ++k) short_pair(A, xi, yi, zi, vxi, vyi, vzi, ri, A.indices[k], s);
    }
    short_store(A, i, s);
}

__global__ void __launch_bounds__(256) k_short_long_rows(const ShortArgs A, const int* __restrict__ queue) {
    const int lane = threadIdx.x & 31;
    const int nq = queue[0];
    for (int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; w < nq; w += (gridDim.x * blockDim.x) >> 5) {
        const long long i = queue[1 + w];
        const long long b = A.offsets[i], e = A.offsets[i + 1];
        const double xi = A.x[i], yi = A.y[i], zi = A.z[i], vxi = A.vx[i], vyi = A.vy[i], vzi = A.vz[i], ri = A.rout[i];
        Sum7 s = {0, 0, 0, 0, 0, 0, 0};
        for (long long k = b + lane; k < e; k += 32) short_pair(A, xi, yi, zi, vxi, vyi, vzi, ri, A.indices[k], s);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            s.a0 += __shfl_down_sync(0xffffffffu, s.a0, o); s.a1 += __shfl_down_sync(0xffffffffu, s.a1, o); s.a2 += __shfl_down_sync(0xffffffffu, s.a2, o);
            s.j0 += __shfl_down_sync(0xffffffffu, s.j0, o); s.j1 += __shfl_down_sync(0xffffffffu, s.j1, o); s.j2 += __shfl_down_sync(0xffffffffu, s.j2, o);
            s.p += __shfl_down_sync(0xffffffffu, s.p, o);
        }
        if (lane == 0) short_store(A, i, s);
    }
}

static size_t short_queue_bytes(int64_t N) { return ((size_t)(N + 1) * 4 + 255) / 256 * 256; }
extern "C" size_t petar_short_range_workspace_bytes(int64_t N) { return N < 0 ? 0 : short_queue_bytes(N) + (size_t)N * sizeof(ShortRec); }

extern "C" int petar_short_range_force(const double* x, const double* y, const double* z, const double* vx, const double* vy, const double* vz,
                                       const double* m, const double* r_out, const int64_t* offsets, const int32_t* indices, int64_t N,
                                       double G, double r_in_over_r_out, double* acc_x, double* acc_y, double* acc_z,
                                       double* jerk_x, double* jerk_y, double* jerk_z, double* pot,
                                       void* workspace, size_t workspace_bytes, void* cuda_stream) {
    if (N < 0 || N > 2000000000ll || !(r_in_over_r_out > 0.0 && r_in_over_r_out < 1.0) || !(G == G)) return PETAR_EINVAL;
    if (N == 0) return PETAR_OK;
    if (!x || !y || !z || !vx || !vy || !vz || !m || !r_out || !offsets) return PETAR_EINVAL;
    if (!workspace || workspace_bytes < petar_short_range_workspace_bytes(N) || ((uintptr_t)workspace & 255u)) return PETAR_EWORKSPACE;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    ShortArgs A;
    A.x = x; A.y = y; A.z = z; A.vx = vx; A.vy = vy; A.vz = vz; A.m = m; A.rout = r_out;
    A.offsets = (const long long*)offsets; A.indices = indices;
    A.ax = acc_x; A.ay = acc_y; A.az = acc_z; A.jx = jerk_x; A.jy = jerk_y; A.jz = jerk_z; A.pot = pot;
    A.G = G; A.rho = r_in_over_r_out; A.lam = (1.0 - r_in_over_r_out) / (1.0 + r_in_over_r_out);
    A.q = r_in_over_r_out / (1.0 - r_in_over_r_out); A.n = N;
    int* queue = (int*)workspace;
    ShortRec* rec = (ShortRec*)((char*)workspace + short_queue_bytes(N));
    A.rec = rec;
    if (cudaMemsetAsync(queue, 0, 4, s) != cudaSuccess) return PETAR_ECUDA;
    k_short_pack<<<cdiv(N, 256), 256, 0, s>>>(A, rec);
    KCHECK(s, "k_short_pack");
    k_short_rows<<<cdiv(N, 256), 256, 0, s>>>(A, queue);
    KCHECK(s, "k_short_rows");
    k_short_long_rows<<<sm_count() * 4, 256, 0, s>>>(A, queue);
    KCHECK(s, "k_short_long_rows");
    petar_count_launch(3);
    return cudaGetLastError() == cudaSuccess ? PETAR_OK : PETAR_ECUDA;
}

// ---- petar_short_range_force_noalloc: the same three kernels for callers that have no way to allocate ------------
// petar_short_range_force needs 68 bytes of caller-supplied device workspace per particle.  Some callers cannot
// supply any: a plug-in that is handed device pointers by a host program and owns no allocator; a step that runs inside
// somebody else's memory pool whose budget is already spent; a real-time or stream-ordered loop in which a
// cudaMalloc (which synchronises the whole device) is not acceptable.  For them the workspace below is part of the
// library image: a fixed array in device global memory, PETAR_SHORT_RANGE_NOALLOC_MAX_N particles large (about
// 4.3 MB).  Every GPU on which this library's code is loaded carries that array until the process exits,
// whether or not the entry point is ever called -- which is why the limit is small.
#define NOALLOC_QUEUE_BYTES ((((size_t)PETAR_SHORT_RANGE_NOALLOC_MAX_N + 1) * 4 + 255) / 256 * 256)
#define NOALLOC_BYTES (NOALLOC_QUEUE_BYTES + (size_t)PETAR_SHORT_RANGE_NOALLOC_MAX_N * sizeof(ShortRec))
static __device__ __align__(256) unsigned char g_short_noalloc_scratch[NOALLOC_BYTES];

// In HOST code the name g_short_noalloc_scratch is only the handle by which the runtime knows the array; it is not
// the array's address on the GPU and must never be handed to a kernel.  The address is asked for once per device
// (with that device current) and remembered; devices beyond the table are looked up on every call.
#define NOALLOC_MAX_DEVICES 64
static void* g_noalloc_ptr[NOALLOC_MAX_DEVICES];
static std::mutex g_noalloc_mutex;

static cudaError_t noalloc_scratch(void** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool cached = dev >= 0 && dev < NOALLOC_MAX_DEVICES;
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (cached && g_noalloc_ptr[dev]) { *out = g_noalloc_ptr[dev]; return cudaSuccess; }
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_short_noalloc_scratch);
    if (e != cudaSuccess) return e;
    if (!p || ((uintptr_t)p & 255u)) return cudaErrorInvalidSymbol;
    if (cached) g_noalloc_ptr[dev] = p;
    *out = p;
    return cudaSuccess;
}

extern "C" int petar_short_range_force_noalloc(const double* x, const double* y, const double* z, const double* vx, const double* vy,
                                               const double* vz, const double* m, const double* r_out, const int64_t* offsets,
                                               const int32_t* indices, int64_t N, double G, double r_in_over_r_out,
                                               double* acc_x, double* acc_y, double* acc_z, double* jerk_x, double* jerk_y,
                                               double* jerk_z, double* pot, void* cuda_stream) {
    if (N < 0 || !(r_in_over_r_out > 0.0 && r_in_over_r_out < 1.0) || !(G == G)) return PETAR_EINVAL;
    if (N > PETAR_SHORT_RANGE_NOALLOC_MAX_N) return PETAR_ECAPACITY;          // before anything is touched or enqueued
    if (N == 0) return PETAR_OK;
    if (!x || !y || !z || !vx || !vy || !vz || !m || !r_out || !offsets) return PETAR_EINVAL;
    void* scratch = nullptr;
    if (noalloc_scratch(&scratch) != cudaSuccess) return PETAR_ECUDA;         // first call on this device: the set-up
    cudaStream_t s = (cudaStream_t)cuda_stream;
    ShortArgs A;
    A.x = x; A.y = y; A.z = z; A.vx = vx; A.vy = vy; A.vz = vz; A.m = m; A.rout = r_out;
    A.offsets = (const long long*)offsets; A.indices = indices;
    A.ax = acc_x; A.ay = acc_y; A.az = acc_z; A.jx = jerk_x; A.jy = jerk_y; A.jz = jerk_z; A.pot = pot;
    A.G = G; A.rho = r_in_over_r_out; A.lam = (1.0 - r_in_over_r_out) / (1.0 + r_in_over_r_out);
    A.q = r_in_over_r_out / (1.0 - r_in_over_r_out); A.n = N;
    // same split of the scratch as the workspace of petar_short_range_force, at the fixed maximum size
    int* queue = (int*)scratch;
    ShortRec* rec = (ShortRec*)((char*)scratch + NOALLOC_QUEUE_BYTES);
    A.rec = rec;
    // The array still holds what the previous call left.  Only the long-row counter queue[0] has to start at zero;
    // the records and queue entries that this call reads are all written by this call first.
    if (cudaMemsetAsync(queue, 0, 4, s) != cudaSuccess) return PETAR_ECUDA;
    k_short_pack<<<cdiv(N, 256), 256, 0, s>>>(A, rec);
    KCHECK(s, "k_short_pack");
    k_short_rows<<<cdiv(N, 256), 256, 0, s>>>(A, queue);
    KCHECK(s, "k_short_rows");
    k_short_long_rows<<<sm_count() * 4, 256, 0, s>>>(A, queue);
    KCHECK(s, "k_short_long_rows");
    petar_count_launch(3);
    return cudaGetLastError() == cudaSuccess ? PETAR_OK : PETAR_ECUDA;
}

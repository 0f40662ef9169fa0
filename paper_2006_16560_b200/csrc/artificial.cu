// artificial.cu -- SURVEY.md 8(f) rank 3: the steps either side of the long-range force.
//   petar_kick                 : P3T-kick  v += a_L dt
//   petar_artificial_particles : per binary, the tidal-tensor measure points (Table 1 part (3)),
//                                the centre-of-mass point and the three pseudoparticles of Eq. 38 (:473-478) that
//                                carry the orbit-averaged quadrupole of Eq. 36-37
//   petar_tidal_tensor_fit     : coefficients of Eq. 25-26 from the accelerations measured at those points, with
//                                the generalized inverse of Eq. 28 (tidal_tables.inc, generated; equals Table 1)
// One thread per binary, fp64.  Readings P24-P26 of DESIGN.md.
#include "internal.cuh"
#include "tidal_tables.inc"

__global__ void __launch_bounds__(256) k_kick(double* __restrict__ vx, double* __restrict__ vy, double* __restrict__ vz,
                                              const double* __restrict__ ax, const double* __restrict__ ay, const double* __restrict__ az,
                                              double dt, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    vx[i] = vx[i] + ax[i] * dt; vy[i] = vy[i] + ay[i] * dt; vz[i] = vz[i] + az[i] * dt;
}

extern "C" int petar_kick(double* vx, double* vy, double* vz, const double* ax, const double* ay, const double* az, double dt,
                          int64_t N, void* cuda_stream) {
    if (N < 0 || !(dt == dt)) return PETAR_EINVAL;
    if (N == 0) return PETAR_OK;
    if (!vx || !vy || !vz || !ax || !ay || !az) return PETAR_EINVAL;
    k_kick<<<cdiv(N, 256), 256, 0, (cudaStream_t)cuda_stream>>>(vx, vy, vz, ax, ay, az, dt, N);
    petar_count_launch(1);
    return cudaGetLastError() == cudaSuccess ? PETAR_OK : PETAR_ECUDA;
}

// Kepler elements and orbital frame of a pair (reading P26): P to the pericentre, Q = W x P, W along d x w
struct BinFrame { double a, e, inv_a, mt, cm[3], P[3], Q[3]; bool bound; };
__device__ __forceinline__ BinFrame binary_frame(const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
                                                 const double* __restrict__ vx, const double* __restrict__ vy, const double* __restrict__ vz,
                                                 const double* __restrict__ m, const int i1, const int i2, const double G) {
    BinFrame f;
    const double m1 = m[i1], m2 = m[i2];
    f.mt = m1 + m2;
    const double x1[3] = {x[i1], y[i1], z[i1]}, x2[3] = {x[i2], y[i2], z[i2]};
    const double d[3] = {x2[0] - x1[0], x2[1] - x1[1], x2[2] - x1[2]};
    const double w[3] = {vx[i2] - vx[i1], vy[i2] - vy[i1], vz[i2] - vz[i1]};
    for (int k = 0; k < 3; ++k) f.cm[k] = (m1 * x1[k] + m2 * x2[k]) / f.mt;
    const double mu = G * f.mt;
    const double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    const double v2 = w[0] * w[0] + w[1] * w[1] + w[2] * w[2];
    const double h[3] = {d[1] * w[2] - d[2] * w[1], d[2] * w[0] - d[0] * w[2], d[0] * w[1] - d[1] * w[0]};
    const double hn = sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]);
    f.inv_a = 2.0 / r - v2 / mu;
    // eccentricity vector (w x h) / mu - d / r
    const double ev[3] = {(w[1] * h[2] - w[2] * h[1]) / mu - d[0] / r, (w[2] * h[0] - w[0] * h[2]) / mu - d[1] / r, (w[0] * h[1] - w[1] * h[0]) / mu - d[2] / r};
    f.e = sqrt(ev[0] * ev[0] + ev[1] * ev[1] + ev[2] * ev[2]);
    f.bound = f.inv_a > 0.0 && hn > 0.0;
    f.a = f.bound ? 1.0 / f.inv_a : 0.0;
    for (int k = 0; k < 3; ++k) { f.P[k] = k == 0; f.Q[k] = k == 1; }
    if (f.bound) {
        const double W[3] = {h[0] / hn, h[1] / hn, h[2] / hn};
        if (f.e > 1e-12) { f.P[0] = ev[0] / f.e; f.P[1] = ev[1] / f.e; f.P[2] = ev[2] / f.e; } else { f.P[0] = d[0] / r; f.P[1] = d[1] / r; f.P[2] = d[2] / r; }
        const double pw = f.P[0] * W[0] + f.P[1] * W[1] + f.P[2] * W[2];
        for (int k = 0; k < 3; ++k) f.P[k] -= W[k] * pw;
        const double pn = sqrt(f.P[0] * f.P[0] + f.P[1] * f.P[1] + f.P[2] * f.P[2]);
        for (int k = 0; k < 3; ++k) f.P[k] /= pn;
        f.Q[0] = W[1] * f.P[2] - W[2] * f.P[1]; f.Q[1] = W[2] * f.P[0] - W[0] * f.P[2]; f.Q[2] = W[0] * f.P[1] - W[1] * f.P[0];
    }
    return f;
}

struct ArtArgs {
    const double *x, *y, *z, *vx, *vy, *vz, *m;
    const int* pairs;
    double *ox, *oy, *oz, *om, *elem;
    double G, tt_scale;
    long long nb;
    int order;
};

__global__ void __launch_bounds__(128) k_artificial(const ArtArgs A) {
    const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= A.nb) return;
    const int i1 = A.pairs[2 * b], i2 = A.pairs[2 * b + 1];
    const double m1 = A.m[i1], m2 = A.m[i2];
    const BinFrame f = binary_frame(A.x, A.y, A.z, A.vx, A.vy, A.vz, A.m, i1, i2, A.G);
    const double mt = f.mt, e = f.e, a = f.a, inv_a = f.inv_a;
    const bool bound = f.bound;
    const double* cm = f.cm;
    const int ntt = A.order == 2 ? 4 : 8;
    const int na = ntt + 4;
    double* ox = A.ox + b * na; double* oy = A.oy + b * na; double* oz = A.oz + b * na; double* om = A.om + b * na;
    for (int k = 0; k < na; ++k) { ox[k] = cm[0]; oy[k] = cm[1]; oz[k] = cm[2]; om[k] = k > ntt ? mt / 3.0 : 0.0; }
    double d_c = 0.0;
    if (bound) {
        d_c = A.tt_scale * a;
        for (int k = 0; k < ntt; ++k) {
            const double* p = A.order == 2 ? c_tt_points2[k] : c_tt_points3[k];
            ox[k] = cm[0] + d_c * p[0]; oy[k] = cm[1] + d_c * p[1]; oz[k] = cm[2] + d_c * p[2];
        }
        // Eq. 38
        const double s = a * sqrt((m1 * m2 / mt) / mt);
        const double bx = sqrt(3.0 * e * e + 0.75), by = sqrt(1.0 - e * e);
        const double lx[3] = {0.0, s * bx, -s * bx}, ly[3] = {s * by, -0.5 * s * by, -0.5 * s * by};
        for (int k = 0; k < 3; ++k) {
            ox[ntt + 1 + k] = cm[0] + lx[k] * f.P[0] + ly[k] * f.Q[0];
            oy[ntt + 1 + k] = cm[1] + lx[k] * f.P[1] + ly[k] * f.Q[1];
            oz[ntt + 1 + k] = cm[2] + lx[k] * f.P[2] + ly[k] * f.Q[2];
        }
    }
    if (A.elem) {
        double* el = A.elem + 8 * b;
        el[0] = bound ? a : (inv_a != 0.0 ? 1.0 / inv_a : 0.0); el[1] = e; el[2] = d_c; el[3] = cm[0]; el[4] = cm[1]; el[5] = cm[2];
        el[6] = bound ? 1.0 : 0.0; el[7] = mt;
    }
}

extern "C" int petar_artificial_particles(const double* x, const double* y, const double* z, const double* vx, const double* vy,
                                          const double* vz, const double* m, const int32_t* pairs, int64_t n_bin, double G,
                                          int32_t order, double tt_scale, double* art_x, double* art_y, double* art_z, double* art_m,
                                          double* elem, void* cuda_stream) {
    if (n_bin < 0 || (order != 2 && order != 3) || !(tt_scale > 0.0) || !(G > 0.0)) return PETAR_EINVAL;
    if (n_bin == 0) return PETAR_OK;
    if (!x || !y || !z || !vx || !vy || !vz || !m || !pairs || !art_x || !art_y || !art_z || !art_m) return PETAR_EINVAL;
    ArtArgs A = {x, y, z, vx, vy, vz, m, pairs, art_x, art_y, art_z, art_m, elem, G, tt_scale, n_bin, order};
    k_artificial<<<cdiv(n_bin, 128), 128, 0, (cudaStream_t)cuda_stream>>>(A);
    petar_count_launch(1);
    return cudaGetLastError() == cudaSuccess ? PETAR_OK : PETAR_ECUDA;
}

// Orbit-sampling particles (Eq. 29; reading P27): n_split samples per component at E_k = k dE
__global__ void __launch_bounds__(128) k_orbit_sampling(const ArtArgs A, const int n_split) {
    const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= A.nb) return;
    const int i1 = A.pairs[2 * b], i2 = A.pairs[2 * b + 1];
    const double m1 = A.m[i1], m2 = A.m[i2];
    const BinFrame f = binary_frame(A.x, A.y, A.z, A.vx, A.vy, A.vz, A.m, i1, i2, A.G);
    const double twopi = 6.283185307179586476925;
    const double dE = twopi / (double)n_split, shalf = sin(0.5 * dE), by = sqrt(fmax(0.0, 1.0 - f.e * f.e));
    double* ox = A.ox + b * 2 * n_split; double* oy = A.oy + b * 2 * n_split; double* oz = A.oz + b * 2 * n_split; double* om = A.om + b * 2 * n_split;
    for (int k = 0; k < n_split; ++k) {
        double rel[3] = {0.0, 0.0, 0.0}, dM = dE;
        if (f.bound) {
            double sE, cE;
            sincos((double)k * dE, &sE, &cE);
            dM = dE - 2.0 * f.e * cE * shalf;
            const double lx = f.a * (cE - f.e), ly = f.a * by * sE;                       // Eq. 32
            for (int c = 0; c < 3; ++c) rel[c] = lx * f.P[c] + ly * f.Q[c];
        }
        const double q1 = m2 / f.mt, q2 = m1 / f.mt;                                         // Eq. 33
        ox[k] = f.cm[0] - q1 * rel[0]; oy[k] = f.cm[1] - q1 * rel[1]; oz[k] = f.cm[2] - q1 * rel[2];
        ox[n_split + k] = f.cm[0] + q2 * rel[0]; oy[n_split + k] = f.cm[1] + q2 * rel[1]; oz[n_split + k] = f.cm[2] + q2 * rel[2];
        om[k] = m1 * dM / twopi; om[n_split + k] = m2 * dM / twopi;
    }
}

extern "C" int petar_orbit_sampling(const double* x, const double* y, const double* z, const double* vx, const double* vy,
                                    const double* vz, const double* m, const int32_t* pairs, int64_t n_bin, double G,
                                    int32_t n_split, double* out_x, double* out_y, double* out_z, double* out_m, void* cuda_stream) {
    if (n_bin < 0 || n_split < 1 || n_split > 1024 || !(G > 0.0)) return PETAR_EINVAL;
    if (n_bin == 0) return PETAR_OK;
    if (!x || !y || !z || !vx || !vy || !vz || !m || !pairs || !out_x || !out_y || !out_z || !out_m) return PETAR_EINVAL;
    ArtArgs A = {x, y, z, vx, vy, vz, m, pairs, out_x, out_y, out_z, out_m, nullptr, G, 1.0, n_bin, 2};
    k_orbit_sampling<<<cdiv(n_bin, 128), 128, 0, (cudaStream_t)cuda_stream>>>(A, n_split);
    petar_count_launch(1);
    return cudaGetLastError() == cudaSuccess ? PETAR_OK : PETAR_ECUDA;
}

// T[b][c] = sum_k inv[c][k] A'_k / d_c^(1 or 2),  A' = A(r_k) - A(r_cm)  (Eq. 27-28)
__global__ void __launch_bounds__(128) k_tidal_fit(const double* __restrict__ ax, const double* __restrict__ ay, const double* __restrict__ az,
                                                   const double* __restrict__ elem, long long nb, int order, double* __restrict__ T) {
    const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nb) return;
    const int ntt = order == 2 ? 4 : 8, na = ntt + 4, nc = order == 2 ? 6 : 16;
    const double d_c = elem[8 * b + 2];
    double* out = T + b * nc;
    if (!(d_c > 0.0)) { for (int c = 0; c < nc; ++c) out[c] = 0.0; return; }
    const double acm[3] = {ax[b * na + ntt], ay[b * na + ntt], az[b * na + ntt]};
    double Ap[24];
    for (int k = 0; k < ntt; ++k) { Ap[3 * k] = ax[b * na + k] - acm[0]; Ap[3 * k + 1] = ay[b * na + k] - acm[1]; Ap[3 * k + 2] = az[b * na + k] - acm[2]; }
    const double s1 = 1.0 / d_c, s2 = s1 * s1;
    for (int c = 0; c < nc; ++c) {
        double acc = 0.0;
        for (int k = 0; k < 3 * ntt; ++k) acc += (order == 2 ? c_tt_inv2[c][k] : c_tt_inv3[c][k]) * Ap[k];
        out[c] = acc * (c < 6 ? s1 : s2);
    }
}

extern "C" int petar_tidal_tensor_fit(const double* acc_x, const double* acc_y, const double* acc_z, const double* elem, int64_t n_bin,
                                      int32_t order, double* T, void* cuda_stream) {
    if (n_bin < 0 || (order != 2 && order != 3)) return PETAR_EINVAL;
    if (n_bin == 0) return PETAR_OK;
    if (!acc_x || !acc_y || !acc_z || !elem || !T) return PETAR_EINVAL;
    k_tidal_fit<<<cdiv(n_bin, 128), 128, 0, (cudaStream_t)cuda_stream>>>(acc_x, acc_y, acc_z, elem, n_bin, order, T);
    petar_count_launch(1);
    return cudaGetLastError() == cudaSuccess ? PETAR_OK : PETAR_ECUDA;
}

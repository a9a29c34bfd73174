// fit.cu -- circle fit of the hits assigned to each kept candidate ("further computations (e.g., a full
// Kalman fit) ... obtain the best measurement of the track parameters"; reading D11: an algebraic
// Kasa circle fit in double precision stands in for the Kalman fit).
//   K-fit-a  zero the moment rows of the candidates in use
//   K-fit-b  one thread per hit: 9 double atomicAdds {n, Sx, Sy, Sz, Sxx, Sxy, Syy, Sxz, Syz} into its candidate's row
//   K-fit-c  one thread per candidate: 3x3 normal equations by Cramer's rule, centre / radius, D1 parameters
#include <cmath>

#include "common.cuh"

namespace {

__global__ void __launch_bounds__(256) fit_zero_kernel(const int32_t* __restrict__ cand_off, int n_events, int capacity,
                                                       double* __restrict__ work) {
    const int n_c = min(cand_off[n_events], capacity);
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t < (long long)n_c * 9) work[t] = 0.0;
}

__global__ void __launch_bounds__(256) fit_moments_kernel(const float2* __restrict__ hits, int n_hits,
                                                          const int32_t* __restrict__ hit_to_cand,
                                                          const int32_t* __restrict__ cand_off, int n_events, int capacity,
                                                          double* __restrict__ work) {
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= n_hits) return;
    const int c = hit_to_cand[h];
    if (c < 0 || c >= min(cand_off[n_events], capacity)) return;
    const float2 p = __ldg(hits + h);
    const double x = (double)p.x, y = (double)p.y;
    const double z = x * x + y * y;
    double* a = work + (size_t)c * 9;
    atomicAdd(a + 0, 1.0); atomicAdd(a + 1, x); atomicAdd(a + 2, y); atomicAdd(a + 3, z);
    atomicAdd(a + 4, x * x); atomicAdd(a + 5, x * y); atomicAdd(a + 6, y * y); atomicAdd(a + 7, x * z); atomicAdd(a + 8, y * z);
}

__global__ void __launch_bounds__(128) fit_solve_kernel(HoughConsts c, double kb, const hough_candidate* __restrict__ cands,
                                                        const int32_t* __restrict__ cand_off, int n_events, int capacity,
                                                        const uint8_t* __restrict__ keep, const double* __restrict__ work,
                                                        hough_track_fit* __restrict__ fit, int32_t* __restrict__ n_fit) {
    const int ci = blockIdx.x * blockDim.x + threadIdx.x;
    if (ci >= capacity) return;
    hough_track_fit f;
    f.phi0 = f.qpt = f.d0 = f.radius = 0.0;
    int nf = 0;
    const int n_c = min(cand_off[n_events], capacity);
    if (ci < n_c && (!keep || keep[ci])) {
        const double* a = work + (size_t)ci * 9;
        const double n = a[0], Sx = a[1], Sy = a[2], Sz = a[3], Sxx = a[4], Sxy = a[5], Syy = a[6], Sxz = a[7], Syz = a[8];
        const int ni = (int)n;
        nf = -ni;
        if (ni >= 3) {
            const double det = Sxx * (Syy * n - Sy * Sy) - Sxy * (Sxy * n - Sy * Sx) + Sx * (Sxy * Sy - Syy * Sx);
            if (fabs(det) > 1.0e-9 * fabs(Sxx * Syy * n)) {
                const double r1 = -Sxz, r2 = -Syz, r3 = -Sz;
                const double B = (r1 * (Syy * n - Sy * Sy) - Sxy * (r2 * n - Sy * r3) + Sx * (r2 * Sy - Syy * r3)) / det;
                const double Cc = (Sxx * (r2 * n - r3 * Sy) - r1 * (Sxy * n - Sy * Sx) + Sx * (Sxy * r3 - r2 * Sx)) / det;
                const double D = (Sxx * (Syy * r3 - Sy * r2) - Sxy * (Sxy * r3 - r2 * Sx) + r1 * (Sxy * Sy - Syy * Sx)) / det;
                const double xc = -0.5 * B, yc = -0.5 * Cc;
                const double R2 = xc * xc + yc * yc - D;
                const double cn = sqrt(xc * xc + yc * yc);
                if (R2 > 0.0 && cn > 0.0) {
                    const double R = sqrt(R2);
                    const double theta = ((double)cands[ci].i + 0.5) * (2.0 * 3.14159265358979323846 / (double)c.n_phi);
                    double tx = -yc / cn, ty = xc / cn;
                    if (tx * cos(theta) + ty * sin(theta) < 0.0) { tx = -tx; ty = -ty; }
                    const double s = 1.0 - R / cn;
                    const double p0x = xc * s, p0y = yc * s;
                    const double nx = -ty, ny = tx;
                    double phi0 = atan2(ty, tx);
                    if (phi0 < 0.0) phi0 += 2.0 * 3.14159265358979323846;
                    const double inv_rho = (xc - p0x) * nx + (yc - p0y) * ny;
                    f.phi0 = phi0;
                    f.qpt = (kb != 0.0) ? -(1.0 / inv_rho) / kb : 0.0;
                    f.d0 = p0x * nx + p0y * ny;
                    f.radius = R;
                    nf = ni;
                }
            }
        }
    }
    fit[ci] = f;
    n_fit[ci] = nf;
}

}  // namespace

extern "C" int hough_fit_circles(hough_plan* p, const float* d_hits_xy, int32_t n_hits, const int32_t* d_hit_to_cand,
                                 const hough_candidate* d_cands, const int32_t* d_cand_offsets, int32_t n_events,
                                 int32_t capacity, const uint8_t* d_cand_keep, double* d_work, hough_track_fit* d_fit,
                                 int32_t* d_n_fit, void* cuda_stream) {
    if (!p || !d_cand_offsets) return HOUGH_ERR_INVALID_ARG;
    if (n_hits < 0 || n_events < 0 || capacity < 0) return HOUGH_ERR_INVALID_ARG;
    if (n_hits > 0 && (!d_hits_xy || !d_hit_to_cand)) return HOUGH_ERR_INVALID_ARG;
    if (capacity > 0 && (!d_cands || !d_work || !d_fit || !d_n_fit)) return HOUGH_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(d_hits_xy) & 7u) || (reinterpret_cast<uintptr_t>(d_cands) & 15u) ||
        (reinterpret_cast<uintptr_t>(d_work) & 7u) || (reinterpret_cast<uintptr_t>(d_fit) & 7u))
        return HOUGH_ERR_INVALID_ARG;
    if (capacity == 0) return HOUGH_OK;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const long long cells = (long long)capacity * 9;
    fit_zero_kernel<<<(unsigned)((cells + 255) / 256), 256, 0, st>>>(d_cand_offsets, n_events, capacity, d_work);
    HOUGH_CUDA_TRY(cudaGetLastError());
    if (n_hits > 0) {
        fit_moments_kernel<<<(n_hits + 255) / 256, 256, 0, st>>>(reinterpret_cast<const float2*>(d_hits_xy), n_hits,
                                                                 d_hit_to_cand, d_cand_offsets, n_events, capacity, d_work);
        HOUGH_CUDA_TRY(cudaGetLastError());
    }
    const double kb = 0.00299792458 * (double)p->bz;
    fit_solve_kernel<<<(capacity + 127) / 128, 128, 0, st>>>(p->c, kb, d_cands, d_cand_offsets, n_events, capacity, d_cand_keep,
                                                            d_work, d_fit, d_n_fit);
    HOUGH_CUDA_TRY(cudaGetLastError());
    hough_count_launches(n_hits > 0 ? 3 : 2);
    return HOUGH_OK;
}

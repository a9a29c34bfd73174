// fit.cu -- circle fit of the hits assigned to each kept candidate ("further computations (e.g., a full
// Kalman fit) ... obtain the best measurement of the track parameters"; reading D11: an algebraic
// Kasa circle fit in double precision stands in for the Kalman fit).
//   K-fit-a  zero the moment rows of the candidates that will be fitted (kept ones, or all without keep flags)
//   K-fit-b  one thread per hit: 9 double atomicAdds {n, Sx, Sy, Sz, Sxx, Sxy, Syy, Sxz, Syz} into its candidate's row
//   K-fit-c  one thread per candidate: moments about the hits' centroid, 2x2 solve for the centre, D1 parameters in
//            closed form from (centre, R, orientation) -- a different algebraic route from the 3x3 Cramer solve of the CPU
//            checker under tests/, so that the parity test compares two independent solves
#include <algorithm>
#include <cmath>
#include <mutex>

#include "common.cuh"

namespace {

// K-fit-a: one thread per candidate row (grid-stride over a fixed grid: the list length is only known on the device), and
// only the rows that will be read -- of 6.6 M candidates per 256-event call of config 3, 48 k are kept.
__global__ void __launch_bounds__(256) fit_zero_kernel(const int32_t* __restrict__ cand_off, int n_events, int capacity,
                                                       const uint8_t* __restrict__ keep, double* __restrict__ work) {
    const int n_c = min(cand_off[n_events], capacity);
    for (long long ci = (long long)blockIdx.x * blockDim.x + threadIdx.x; ci < n_c; ci += (long long)gridDim.x * blockDim.x) {
        if (keep && !keep[ci]) continue;
        double* a = work + (size_t)ci * 9;
#pragma unroll
        for (int q = 0; q < 9; ++q) a[q] = 0.0;
    }
}

__global__ void __launch_bounds__(256) fit_moments_kernel(const float2* __restrict__ hits, int n_hits,
                                                          const int32_t* __restrict__ hit_to_cand,
                                                          const int32_t* __restrict__ cand_off, int n_events, int capacity,
                                                          const uint8_t* __restrict__ keep, double* __restrict__ work) {
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= n_hits) return;
    const int c = hit_to_cand[h];
    if (c < 0 || c >= min(cand_off[n_events], capacity)) return;
    if (keep && !keep[c]) return;                            // that row was not zeroed and will not be read
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
        // Raw sums of the candidate's hits: m0 = count, m1 = (Sx, Sy), Sz = sum |p|^2, second moments, and sum p |p|^2.
        const double* a = work + (size_t)ci * 9;
        const double m0 = a[0];
        const int cnt = (int)m0;
        nf = -cnt;
        if (cnt >= 3) {
            // Work about the centroid g = m1 / m0 (u = p - g).  Centred second moments and the centred cubic sums
            // T = sum u |u|^2 follow from the raw sums; the Kasa minimum has its centre at g + c with
            //     [Cuu Cuv; Cuv Cvv] c = T / 2        and       R^2 = |c|^2 + (Cuu + Cvv) / m0.
            const double gx = a[1] / m0, gy = a[2] / m0, gg = gx * gx + gy * gy;
            const double Cuu = a[4] - gx * a[1], Cuv = a[5] - gx * a[2], Cvv = a[6] - gy * a[2];
            const double zc = a[3] - 2.0 * (gx * a[1] + gy * a[2]) + m0 * gg;                      // sum |u|^2 = Cuu + Cvv
            const double Tu = a[7] - 2.0 * (gx * a[4] + gy * a[5]) + gg * a[1] - gx * zc;
            const double Tv = a[8] - 2.0 * (gx * a[5] + gy * a[6]) + gg * a[2] - gy * zc;
            const double dd = Cuu * Cvv - Cuv * Cuv;                     // (3x3 normal-equation determinant) / m0
            if (fabs(dd) > 1.0e-9 * fabs(a[4] * a[6])) {                 // D11's singularity test, divided by m0
                const double cu = 0.5 * (Tu * Cvv - Tv * Cuv) / dd, cv = 0.5 * (Tv * Cuu - Tu * Cuv) / dd;
                const double ox = gx + cu, oy = gy + cv;                // circle centre
                const double rr = cu * cu + cv * cv + zc / m0;
                const double oc = hypot(ox, oy);
                if (rr > 0.0 && oc > 0.0) {
                    // D1: the centre is (d0 + 1/rho) n_hat with n_hat = (-sin phi0, cos phi0).  Of the two orientations
                    // n_hat = +-centre/|centre| take the one whose direction of travel (n_y, -n_x) points along the
                    // candidate's column; then 1/rho = s R (|d0| < R), d0 = s (|centre| - R).
                    const double rad = sqrt(rr);
                    double sn, cs;
                    sincos(((double)cands[ci].i + 0.5) * (6.283185307179586476925 / (double)c.n_phi), &sn, &cs);
                    const double s = (oy * cs - ox * sn) >= 0.0 ? 1.0 : -1.0;
                    double ph = atan2(-s * ox, s * oy);
                    if (ph < 0.0) ph += 6.283185307179586476925;
                    f.phi0 = ph;
                    f.qpt = kb != 0.0 ? -s / (rad * kb) : 0.0;
                    f.d0 = s * (oc - rad);
                    f.radius = rad;
                    nf = cnt;
                }
            }
        }
    }
    fit[ci] = f;
    n_fit[ci] = nf;
}

inline unsigned fit_zero_blocks(int capacity) { return (unsigned)std::min((capacity + 255) / 256, 148 * 16); }

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
    fit_zero_kernel<<<fit_zero_blocks(capacity), 256, 0, st>>>(d_cand_offsets, n_events, capacity, d_cand_keep, d_work);
    HOUGH_CUDA_TRY(cudaGetLastError());
    if (n_hits > 0) {
        fit_moments_kernel<<<(n_hits + 255) / 256, 256, 0, st>>>(reinterpret_cast<const float2*>(d_hits_xy), n_hits,
                                                                 d_hit_to_cand, d_cand_offsets, n_events, capacity, d_cand_keep,
                                                                 d_work);
        HOUGH_CUDA_TRY(cudaGetLastError());
    }
    const double kb = 0.00299792458 * (double)p->bz;
    fit_solve_kernel<<<(capacity + 127) / 128, 128, 0, st>>>(p->c, kb, d_cands, d_cand_offsets, n_events, capacity, d_cand_keep,
                                                            d_work, d_fit, d_n_fit);
    HOUGH_CUDA_TRY(cudaGetLastError());
    hough_count_launches(n_hits > 0 ? 3 : 2);
    return HOUGH_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// hough_fit_circles_static: the same three kernels, for callers that must not allocate device memory.
//
// Who that is.  (1) Trigger-style event loops (the paper's setting: a fixed time budget per event):
// cudaMalloc / cudaFree take an unbounded time and stall every stream of the device while they run, so such a loop
// may not reach them once it is live.  (2) Plug-ins inside a host application whose GPU memory is entirely managed by
// someone else (a framework's caching pool, an experiment's memory manager with a fixed budget): they are handed
// their input and output buffers and have nowhere to get 72 bytes of moment scratch per candidate from.
//
// The scratch therefore lives in the library image: one fixed array per GPU, reserved when the library's code is loaded
// onto that GPU and held until the process exits (4.5 MiB).  Consequences a caller has to know:
//   * capacity is limited to HOUGH_FIT_STATIC_MAX_CANDIDATES; larger requests are refused, nothing is enqueued;
//   * all calls on one GPU share the array: two calls whose kernels can be in flight at the same time (different streams,
//     or different host threads on different streams) corrupt each other's sums -- keep them on one stream or order them
//     with events; the array also keeps the previous call's sums, which is why K-fit-a zeroes the rows in use every call;
//   * the first call on each GPU looks up the array's device address (set-up, below); make that first call during
//     start-up, on the device the later calls will use, and before any stream capture is begun.
//
// `g_fit_scratch` as written in host code is only a handle for the runtime's symbol table, NOT a device address:
// handing it to a kernel would make the kernel read and write through a host pointer.  fit_static_scratch() turns it into
// the real address with cudaGetSymbolAddress, per device, because every GPU holds its own copy at its own address.
constexpr int FIT_STATIC_ROW = 9;   // doubles per candidate: {n, Sx, Sy, Sz, Sxx, Sxy, Syy, Sxz, Syz}
static __device__ __align__(256) double g_fit_scratch[(size_t)HOUGH_FIT_STATIC_MAX_CANDIDATES * FIT_STATIC_ROW];

namespace {

std::mutex g_fit_static_mu;
double* g_fit_static_ptr[HOUGH_MAX_DEVICES];   // per device: address of that GPU's copy of g_fit_scratch (null: not looked up)

// Address of the CURRENT device's scratch array.  Cached per device; a device index beyond the cache asks every time.
int fit_static_scratch(double** out) {
    int dev = -1;
    HOUGH_CUDA_TRY(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lock(g_fit_static_mu);
    if (dev >= 0 && dev < HOUGH_MAX_DEVICES && g_fit_static_ptr[dev]) {
        *out = g_fit_static_ptr[dev];
        return HOUGH_OK;
    }
    double* ptr = nullptr;
    HOUGH_CUDA_TRY(cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_fit_scratch));
    if (!ptr) return HOUGH_ERR_CUDA;
    if (dev >= 0 && dev < HOUGH_MAX_DEVICES) g_fit_static_ptr[dev] = ptr;
    *out = ptr;
    return HOUGH_OK;
}

}  // namespace

extern "C" int hough_fit_circles_static(int32_t n_phi, float bz_tesla, const float* d_hits_xy, int32_t n_hits,
                                        const int32_t* d_hit_to_cand, const hough_candidate* d_cands,
                                        const int32_t* d_cand_offsets, int32_t n_events, int32_t capacity,
                                        const uint8_t* d_cand_keep, hough_track_fit* d_fit, int32_t* d_n_fit,
                                        void* cuda_stream) {
    if (!d_cand_offsets || n_phi <= 0) return HOUGH_ERR_INVALID_ARG;
    if (n_hits < 0 || n_events < 0 || capacity < 0) return HOUGH_ERR_INVALID_ARG;
    if (capacity > HOUGH_FIT_STATIC_MAX_CANDIDATES) return HOUGH_ERR_TOO_LARGE;   // the fixed scratch has no more rows
    if (n_hits > 0 && (!d_hits_xy || !d_hit_to_cand)) return HOUGH_ERR_INVALID_ARG;
    if (capacity > 0 && (!d_cands || !d_fit || !d_n_fit)) return HOUGH_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(d_hits_xy) & 7u) || (reinterpret_cast<uintptr_t>(d_cands) & 15u) ||
        (reinterpret_cast<uintptr_t>(d_fit) & 7u))
        return HOUGH_ERR_INVALID_ARG;
    if (capacity == 0) return HOUGH_OK;
    double* d_work = nullptr;
    const int rc = fit_static_scratch(&d_work);
    if (rc != HOUGH_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    HoughConsts c{};                   // the solve reads n_phi only (orientation of the circle by the candidate's column)
    c.n_phi = n_phi;
    fit_zero_kernel<<<fit_zero_blocks(capacity), 256, 0, st>>>(d_cand_offsets, n_events, capacity, d_cand_keep, d_work);
    HOUGH_CUDA_TRY(cudaGetLastError());
    if (n_hits > 0) {
        fit_moments_kernel<<<(n_hits + 255) / 256, 256, 0, st>>>(reinterpret_cast<const float2*>(d_hits_xy), n_hits,
                                                                 d_hit_to_cand, d_cand_offsets, n_events, capacity, d_cand_keep,
                                                                 d_work);
        HOUGH_CUDA_TRY(cudaGetLastError());
    }
    const double kb = 0.00299792458 * (double)bz_tesla;
    fit_solve_kernel<<<(capacity + 127) / 128, 128, 0, st>>>(c, kb, d_cands, d_cand_offsets, n_events, capacity, d_cand_keep,
                                                            d_work, d_fit, d_n_fit);
    HOUGH_CUDA_TRY(cudaGetLastError());
    hough_count_launches(n_hits > 0 ? 3 : 2);
    return HOUGH_OK;
}

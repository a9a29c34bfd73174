// common.cuh -- shared declarations of libhough_b200 (sm_100a only).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/hough.h"

#ifndef __CUDA_ARCH__
#define HOUGH_HOST_ONLY 1
#endif

#define HOUGH_CUDA_TRY(expr)                         \
    do {                                             \
        cudaError_t _e = (expr);                     \
        if (_e != cudaSuccess) {                     \
            hough_set_last_cuda_error(_e, #expr);    \
            return HOUGH_ERR_CUDA;                   \
        }                                            \
    } while (0)

// Self-check build (-DHOUGH_CHECKS=1, `python -m paper_1311_2769_b200.build --checks`): device-side asserts on every
// shared-memory address, queue slot and table index the walk and the peak ring compute.  compute-sanitizer is not
// available on the GPU pool this was developed on; the parity suite is run once against this build instead
// (profiles/r2_checks.md).  Compiled out otherwise.
#ifdef HOUGH_CHECKS
#include <cassert>
#define HOUGH_CHECK(cond) assert(cond)
#else
#define HOUGH_CHECK(cond) ((void)0)
#endif

void hough_set_last_cuda_error(cudaError_t e, const char* what);
void hough_count_launches(int n);   // process-wide count of kernel launches issued by the library

// Plan constants passed by value to kernels (D2).
struct HoughConsts {
    int32_t n_phi, n_qpt, n_d0;
    int32_t bins_per_event;       // n_d0 * n_phi * n_qpt
    int32_t words_per_event;      // ceil(bins_per_event / 32)  (peak bitmask)
    int32_t is_u16;
    int32_t model;                // HOUGH_MODEL_HELIX | HOUGH_MODEL_LINE
    float A_f, qmin, inv_wq, nq_f;
    float qpt_min, d0_min;        // centroid (D7)
    float wq, wphi, wd, two_pi_f;
    float kappa, sd2;             // column-pair recurrence of the walk: 4 sin^2(wphi), 2 sin(wphi)  (walk.cuh "Recurrence")
    const float2* cs;             // [n_phi] {cos, sin} of the column centres
    const float4* d0t;            // [n_d0]  {d0c, 2*d0c, d0c^2, 0}
    // work sizing (windows.cu): never changes a result
    int32_t n_class, n_sector, n_keys;   // radius classes, phi sectors, n_keys = n_class * n_sector (class-major)
    float u_scale;                // n_phi / 2pi : column coordinate u = phi * u_scale - 0.5, phi in [0, 2pi)
    float sector_scale;           // n_sector / 2pi
    const float* edge2;           // [n_class] lower r^2 edge of each class (edge2[0] = 0; last class open-ended)
    const int2* win;              // [n_class][n_d0] {bits(lo_off), steps | fwd_safe << 30}
};

constexpr int HOUGH_MAX_CLASSES = 255;
constexpr int HOUGH_MAX_DEVICES = 64;       // per-device caches of kernel attributes (a device index beyond it: set every call)
constexpr int HOUGH_SECTORS_MIN = 32, HOUGH_SECTORS_MAX = 1024;   // phi sectors of the staging sort: n_phi clamped to this range
constexpr long long HOUGH_STAGE_TABLE_BYTES = 32LL << 20;         // ... and halved until the per-call key-start table fits this

struct HoughWindows {             // host copy of the class / window tables
    int n_class = 0;
    std::vector<float> edge2;     // [n_class]
    std::vector<float> lo_off;    // [n_class * n_d0]
    std::vector<int> steps;       // [n_class * n_d0]
    std::vector<char> fwd_safe;   // [n_class * n_d0] 1: the D3 forward test passes at every column of the window
};
int hough_build_windows(const hough_binning& b, float bz, int n_layers, const float* layer_r, HoughWindows& out);

struct hough_plan {
    hough_binning b;
    float bz;
    int32_t max_hits, max_events;
    int device, sm_count;
    int fullscan;
    int peaks_tiled;                   // 1: find_peaks uses the shared-memory halo-tile kernels instead of the slice walk
    int peaks_regs;                    // 1: 16-bit packed peak walk with register-held rows instead of the cp.async ring
    int peaks_scalar;                  // 1: 16-bit accumulators use the unpacked slice-walk peak kernel (bisecting)
    int exact_walk;                    // 1: the walks evaluate the D3 sequence at every column (no fast path)
    float m_scale;                     // 1 (self-check build: HOUGH_DEBUG_M_SCALE scales the fast path's error bound, to probe its margin)
    int assign_candidates;             // 1: hough_assign_hits takes the candidate-centric path (assoc.cu) instead of re-walking the vote columns
    int reuse_staging;                 // 1: hough_assign_hits may reuse the staging of the preceding hough_vote (same arguments)
    const void* staged_hits; const void* staged_off; int32_t staged_n_hits, staged_n_events; cudaStream_t staged_stream;
    HoughConsts c;
    // geometry (work sizing only)
    int32_t n_layers;
    float layer_r[64];
    // device tables
    float2* d_cs;
    float4* d_d0t;
    // workspace: peaks
    int32_t peak_blocks_per_event;     // blocks of PEAK_BLOCK_BINS bins
    int32_t* d_peak_block_cnt;         // [max_events * peak_blocks_per_event] counts, scanned in place per event
    int32_t* d_event_cnt;              // [max_events + 1]
    uint32_t* d_mask;                  // [max_events * words_per_event] peak bitmask (find_peaks) / candidate bitmask (assign)
    int32_t* d_word_rank;              // [max_events * words_per_event] rank of the first set bit of each word
    unsigned long long* d_best_key;    // [max_hits]
    int2* d_slice;                     // [slice_len] candidate range of each assign tile
    size_t slice_len;
    // device tables: radius classes and column windows (windows.cu)
    float* d_edge2;                    // [n_class]
    int2* d_win;                       // [n_class][n_d0] {bits(lo_off), steps}
    // workspace: staged hits (K1, stage.cu)
    float4* d_staged;                  // [max_hits] {x, y, u, bitcast(original index)} sorted by (event, class, sector)
    int2* d_stage_tmp;                 // [max_hits] {key, rank within key}
    int32_t* d_stage_cnt;              // [max_events][n_keys + 1] key counters -> exclusive key starts
    // candidate-centric association (assoc.cu)
    float2* d_assoc_tab;               // [n_class][n_d0][n_qpt + 1] azimuth-offset hulls per bin edge; null: not built
    int reassign_walk;                 // 1: hough_reassign_hits re-walks the vote columns instead of the candidate-centric path
    int assoc_tab_tried;               // the assoc table was requested once (it may not fit: d_assoc_tab stays null)
    int assoc_tab_borrowed;            // d_assoc_tab belongs to another plan of the same binning / geometry (pipeline lanes): not freed here
    int event_max_steps;               // longest column window of any radius class in slice 0 (work estimate of hough_event_run)
    int event_cluster;                 // 1: hough_event_run takes the cluster kernel whenever it fits, whatever the work estimate says
    int event_general;                 // 1: hough_event_run always takes the three general calls (bisecting / comparison)
    int assoc_smem_configured;         // dynamic shared memory the kernel is configured for on this plan's device
    // vote tile shape (vote.cu)
    int32_t tile32;                    // 1: 32-bit bins in shared memory, 0: two 16-bit bins per word
    int32_t tile_stride_words;         // shared-memory row stride (odd)
    int32_t tile_max_cols;             // phi0 columns per tile that fit the shared-memory budget (0: no tiled path)
};

constexpr int PEAK_BLOCK_BINS = 4096;  // bins per peak-scan block (multiple of 32)

// ---------------------------------------------------------------------------------------------
// D3: the prescribed fp32 vote sequence.  Intrinsics (__f*_rn) are never contracted into FMAs and
// __frcp_rn is the IEEE-correct reciprocal, so the result is independent of compiler flags.
// Returns the q/pT bin or -1.
__device__ __forceinline__ void d3_wf(float x, float y, float c, float s, float& w, float& f) {
    w = __fsub_rn(__fmul_rn(y, c), __fmul_rn(x, s));
    f = __fadd_rn(__fmul_rn(x, c), __fmul_rn(y, s));
}

__device__ __forceinline__ int d3_bin_from_w(float w, float r2, float d0c, float td0, float d0sq, float A_f,
                                             float qmin, float inv_wq, float nq_f, bool line = false) {
    if (line) {                                              // D3L: straight track, the solved parameter is d0 = w
        const float tl = __fmul_rn(__fsub_rn(w, qmin), inv_wq);
        if (!(tl >= 0.0f && tl < nq_f)) return -1;
        return (int)tl;
    }
    const float num = __fsub_rn(d0c, w);
    const float den = __fadd_rn(__fsub_rn(r2, __fmul_rn(td0, w)), d0sq);
    const float g = __fmul_rn(A_f, den);
    const float rinv = __frcp_rn(g);
    const float v = __fmul_rn(num, rinv);
    const float t = __fmul_rn(__fsub_rn(v, qmin), inv_wq);
    if (!(t >= 0.0f && t < nq_f)) return -1;
    return (int)t;
}

__device__ __forceinline__ float d3_r2(float x, float y) { return __fadd_rn(__fmul_rn(x, x), __fmul_rn(y, y)); }

// D7 centroid from the integer moments: every fp32 operation individually rounded.
__device__ __forceinline__ void hough_write_candidate(const HoughConsts& c, hough_candidate* __restrict__ out, int e, int k, int i,
                                                int j, int a, long long S, long long Sj, long long Si, long long Sk) {
    const float fS = __ll2float_rn(S);
    const float oj = __fdiv_rn(__ll2float_rn(Sj), fS);
    const float oi = __fdiv_rn(__ll2float_rn(Si), fS);
    const float ok = __fdiv_rn(__ll2float_rn(Sk), fS);
    const float tj = __fadd_rn(__fadd_rn((float)j, 0.5f), oj);
    const float qpt = __fadd_rn(c.qpt_min, __fmul_rn(tj, c.wq));
    const float ti = __fadd_rn(__fadd_rn((float)i, 0.5f), oi);
    float ph = __fmul_rn(ti, c.wphi);
    if (ph < 0.0f) ph = __fadd_rn(ph, c.two_pi_f);
    else if (ph >= c.two_pi_f) ph = __fsub_rn(ph, c.two_pi_f);
    float d0 = 0.0f;
    if (c.n_d0 > 1) {
        const float tk = __fadd_rn(__fadd_rn((float)k, 0.5f), ok);
        d0 = __fadd_rn(c.d0_min, __fmul_rn(tk, c.wd));
    }
    int4* o = reinterpret_cast<int4*>(out);
    o[0] = make_int4(e, k, i, j);
    o[1] = make_int4(a, __float_as_int(ph), __float_as_int(qpt), __float_as_int(d0));
}

// exclusive scan of n ints in place by one CTA of 1024 threads; the total goes to *total_out.
__device__ __forceinline__ void cta_exclusive_scan(int32_t* data, int n, int32_t* total_out) {
    __shared__ int s_warp[32];
    __shared__ int s_carry;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    for (int base = 0; base < n; base += 1024) {
        const int idx = base + threadIdx.x;
        const int v = idx < n ? data[idx] : 0;
        int x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, x, o);
            if ((threadIdx.x & 31) >= o) x += y;
        }
        if ((threadIdx.x & 31) == 31) s_warp[threadIdx.x >> 5] = x;
        __syncthreads();
        if (threadIdx.x < 32) {
            int ws = s_warp[threadIdx.x];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, ws, o);
                if (threadIdx.x >= o) ws += y;
            }
            s_warp[threadIdx.x] = ws;   // inclusive over warps
        }
        __syncthreads();
        const int warp_prefix = (threadIdx.x >> 5) ? s_warp[(threadIdx.x >> 5) - 1] : 0;
        const int carry = s_carry;
        if (idx < n) data[idx] = carry + warp_prefix + x - v;
        __syncthreads();
        if (threadIdx.x == 0) s_carry = carry + s_warp[31];
        __syncthreads();
    }
    if (threadIdx.x == 0) *total_out = s_carry;
}

// internal entry points (defined in the .cu files)
int hough_stage_hits(hough_plan* p, const float* d_hits_xy, int32_t n_hits, const int32_t* d_event_offsets,
                     int32_t n_events, cudaStream_t st, bool may_reuse);
int hough_build_assoc_table(hough_plan* p);
// Builds the plan's assoc table now if it has none and none was tried (allocates + synchronises: never call it from a
// stream-ordered entry point that may be under capture).  Always HOUGH_OK: a table that does not fit or cannot be built
// leaves d_assoc_tab null, and hough_reassign_hits then re-walks the vote columns.
int hough_prepare_reassign(hough_plan* p);
int hough_assoc_candidates(hough_plan* p, const int32_t* d_event_offsets, int32_t n_hits, int32_t n_events,
                           const hough_candidate* d_cands, const int32_t* d_cand_offsets, int32_t capacity, int32_t assoc_dj,
                           int32_t* d_hit_to_cand, int32_t* d_cand_nhits, cudaStream_t st, const uint8_t* d_keep_filter);
int hough_vote_fullscan(hough_plan* p, const float* d_hits_xy, int32_t n_hits, const int32_t* d_event_offsets,
                        int32_t n_events, void* d_accum, cudaStream_t st);
int hough_vote_tiled(hough_plan* p, const float* d_hits_xy, int32_t n_hits, const int32_t* d_event_offsets,
                     int32_t n_events, void* d_accum, cudaStream_t st);

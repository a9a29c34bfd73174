// stage.cu -- A1: hit staging (B:L5 "a hit-staging kernel that bins hits by phi sector with coalesced,
// vectorised float4 loads"; P:L51 hits are independent).
//
// Per hit: radius class (binary search of r^2 in the plan's class edges), azimuth -> column coordinate u and
// phi sector; counting sort by (event, class, sector) so that 32 consecutive staged hits have the same window
// length and neighbouring columns.  Output record (16 B): {x, y, u, bits(original index within the call)}.
//   K1a stage_count_kernel   : 2 hits per thread (one float4 load), key + rank (atomicAdd on the key counter)
//   K1b stage_scan_kernel    : per event exclusive scan of the key counters (n_keys + 1 entries)
//   K1c stage_scatter_kernel : staged[event_begin + key_start + rank] = record
// The staged order inside a key is whatever the atomics produced; no result depends on it (D4).
#include "common.cuh"

namespace {

__device__ __forceinline__ int find_event_s(const int32_t* __restrict__ off, int n_events, int h) {
    int lo = 0, hi = n_events;          // largest e with off[e] <= h
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (__ldg(off + mid) <= h) lo = mid; else hi = mid;
    }
    return lo;
}

__device__ __forceinline__ void classify(const HoughConsts& c, float x, float y, int& key, float& u) {
    const float r2 = d3_r2(x, y);
    int lo = 0, hi = c.n_class;         // largest class with edge2[class] <= r2; NaN -> last class
    if (!(r2 < __ldg(c.edge2 + c.n_class - 1))) {
        lo = c.n_class - 1;
    } else {
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (__ldg(c.edge2 + mid) <= r2) lo = mid; else hi = mid;
        }
    }
    float phi = atan2f(y, x);
    if (phi < 0.0f) phi += c.two_pi_f;
    if (!(phi >= 0.0f && phi < c.two_pi_f)) phi = 0.0f;       // NaN / rounding at 2pi
    u = phi * c.u_scale - 0.5f;
    int sec = (int)(phi * c.sector_scale);
    sec = min(max(sec, 0), c.n_sector - 1);
    key = lo * c.n_sector + sec;
}

// `hits` is 8-byte aligned (include/hough.h); `lead` = 1 when it is not 16-byte aligned, in which case thread 0
// takes hit 0 alone and every other thread loads the aligned pair (2t - 1, 2t).
__global__ void __launch_bounds__(256) stage_count_kernel(HoughConsts c, const float2* __restrict__ hits, int lead,
                                                          int n_hits, const int32_t* __restrict__ off, int n_events,
                                                          int32_t* __restrict__ key_cnt, int2* __restrict__ tmp) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int h0 = 2 * t - lead;
    if (h0 >= n_hits) return;
    float4 v;
    if (h0 >= 0 && h0 + 1 < n_hits) {
        v = __ldg(reinterpret_cast<const float4*>(hits + h0));
    } else {
        const float2 a = __ldg(hits + (h0 < 0 ? 0 : h0));
        v = h0 < 0 ? make_float4(0.0f, 0.0f, a.x, a.y) : make_float4(a.x, a.y, 0.0f, 0.0f);
    }
    const int e0 = find_event_s(off, n_events, max(h0, 0));
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        const int h = h0 + s;
        if (h < 0) continue;
        if (h >= n_hits) break;
        int e = e0;
        while (e + 1 < n_events && __ldg(off + e + 1) <= h) ++e;     // skip empty events / step to the next one
        int key; float u;
        classify(c, s ? v.z : v.x, s ? v.w : v.y, key, u);
        const int rank = atomicAdd(key_cnt + (size_t)e * (c.n_keys + 1) + key, 1);
        tmp[h] = make_int2(key, rank);
        (void)u;
    }
}

__global__ void __launch_bounds__(1024) stage_scan_kernel(int32_t* __restrict__ key_cnt, int n_keys) {
    __shared__ int32_t total;
    int32_t* row = key_cnt + (size_t)blockIdx.x * (n_keys + 1);
    cta_exclusive_scan(row, n_keys, &total);
    __syncthreads();
    if (threadIdx.x == 0) row[n_keys] = total;
}

__global__ void __launch_bounds__(256) stage_scatter_kernel(HoughConsts c, const float2* __restrict__ hits, int n_hits,
                                                            const int32_t* __restrict__ off, int n_events,
                                                            const int32_t* __restrict__ key_start,
                                                            const int2* __restrict__ tmp, float4* __restrict__ staged) {
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= n_hits) return;
    const float2 p = __ldg(hits + h);
    const int e = find_event_s(off, n_events, h);
    const int2 kr = tmp[h];
    int key; float u;
    classify(c, p.x, p.y, key, u);
    const int pos = __ldg(off + e) + __ldg(key_start + (size_t)e * (c.n_keys + 1) + kr.x) + kr.y;
    staged[pos] = make_float4(p.x, p.y, u, __int_as_float(h));
}

}  // namespace

int hough_stage_hits(hough_plan* p, const float* d_hits_xy, int32_t n_hits, const int32_t* d_event_offsets,
                     int32_t n_events, cudaStream_t st, bool may_reuse) {
    // plan option "reuse_staging": the caller promises that a call with the same pointers, sizes and stream sees the
    // same hits as the previous one (vote followed by assign_hits of one tile), so the staged copy is still valid
    if (may_reuse && p->reuse_staging && p->staged_hits == d_hits_xy && p->staged_off == d_event_offsets && p->staged_n_hits == n_hits &&
        p->staged_n_events == n_events && p->staged_stream == st) {
        p->staged_hits = nullptr;                        // one reuse per staging
        return HOUGH_OK;
    }
    p->staged_hits = d_hits_xy; p->staged_off = d_event_offsets; p->staged_n_hits = n_hits; p->staged_n_events = n_events;
    p->staged_stream = st;
    const size_t cnt_bytes = sizeof(int32_t) * (size_t)n_events * (p->c.n_keys + 1);
    HOUGH_CUDA_TRY(cudaMemsetAsync(p->d_stage_cnt, 0, cnt_bytes, st));
    if (n_hits > 0) {
        const int lead = (reinterpret_cast<uintptr_t>(d_hits_xy) & 15u) ? 1 : 0;
        const int pairs = (n_hits + lead + 1) / 2;
        stage_count_kernel<<<(pairs + 255) / 256, 256, 0, st>>>(p->c, reinterpret_cast<const float2*>(d_hits_xy), lead, n_hits,
                                                                d_event_offsets, n_events, p->d_stage_cnt, p->d_stage_tmp);
        HOUGH_CUDA_TRY(cudaGetLastError());
        hough_count_launches(1);
    }
    stage_scan_kernel<<<n_events, 1024, 0, st>>>(p->d_stage_cnt, p->c.n_keys);
    HOUGH_CUDA_TRY(cudaGetLastError());
    hough_count_launches(1);
    if (n_hits > 0) {
        stage_scatter_kernel<<<(n_hits + 255) / 256, 256, 0, st>>>(p->c, reinterpret_cast<const float2*>(d_hits_xy), n_hits,
                                                                   d_event_offsets, n_events, p->d_stage_cnt,
                                                                   p->d_stage_tmp, p->d_staged);
        HOUGH_CUDA_TRY(cudaGetLastError());
        hough_count_launches(1);
    }
    return HOUGH_OK;
}

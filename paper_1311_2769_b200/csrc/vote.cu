// vote.cu -- A1/A2/A3: hit staging, vote, flush (D3/D4).
#include "walk.cuh"

// ------------------------------------------------------------------------------------------------
// Full-scan reference path (plan option "fullscan" / HOUGH_DEBUG_FULLSCAN=1): one thread per
// (hit, phi0 column), loop over d0 slices, votes straight into global memory with red.add.
// No windowing, no staging: the bisecting path for parity failures.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int find_event(const int32_t* __restrict__ off, int n_events, int h) {
    int lo = 0, hi = n_events;          // largest e with off[e] <= h
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (off[mid] <= h) lo = mid; else hi = mid;
    }
    return lo;
}

template <bool U16>
__global__ void __launch_bounds__(256) vote_fullscan_kernel(HoughConsts c, const float2* __restrict__ hits,
                                                            int n_hits, const int32_t* __restrict__ off,
                                                            int n_events, void* __restrict__ accum) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int h = (int)(t / c.n_phi);
    const int i = (int)(t - (long long)h * c.n_phi);
    if (h >= n_hits) return;
    const float2 p = hits[h];
    const float2 cs = c.cs[i];
    float w, f;
    d3_wf(p.x, p.y, cs.x, cs.y, w, f);
    if (!(f > 0.0f)) return;
    const float r2 = d3_r2(p.x, p.y);
    const int e = find_event(off, n_events, h);
    const size_t ebase = (size_t)e * (size_t)c.bins_per_event;
    for (int k = 0; k < c.n_d0; ++k) {
        const float4 d = c.d0t[k];
        const int j = d3_bin_from_w(w, r2, d.x, d.y, d.z, c.A_f, c.qmin, c.inv_wq, c.nq_f, c.model != 0);
        if (j < 0) continue;
        const size_t bin = ebase + ((size_t)k * c.n_phi + i) * c.n_qpt + j;
        if (U16) {
            atomicAdd(reinterpret_cast<unsigned int*>(accum) + (bin >> 1), 1u << (16 * (unsigned)(bin & 1)));
        } else {
            atomicAdd(reinterpret_cast<int*>(accum) + bin, 1);
        }
    }
}

int hough_vote_fullscan(hough_plan* p, const float* d_hits_xy, int32_t n_hits, const int32_t* d_event_offsets,
                        int32_t n_events, void* d_accum, cudaStream_t st) {
    HOUGH_CUDA_TRY(cudaMemsetAsync(d_accum, 0, hough_accum_bytes(p, n_events), st));
    if (n_hits == 0) return HOUGH_OK;
    const long long threads = (long long)n_hits * p->c.n_phi;
    const long long blocks = (threads + 255) / 256;
    if (blocks > 0x7fffffffLL) return HOUGH_ERR_UNSUPPORTED;
    const float2* hits = reinterpret_cast<const float2*>(d_hits_xy);
    if (p->c.is_u16)
        vote_fullscan_kernel<true><<<(unsigned)blocks, 256, 0, st>>>(p->c, hits, n_hits, d_event_offsets, n_events, d_accum);
    else
        vote_fullscan_kernel<false><<<(unsigned)blocks, 256, 0, st>>>(p->c, hits, n_hits, d_event_offsets, n_events, d_accum);
    HOUGH_CUDA_TRY(cudaGetLastError());
    hough_count_launches(1);
    return HOUGH_OK;
}

// ------------------------------------------------------------------------------------------------
// Tiled path (A1 -> A2 -> A3): stage the hits, then the column walk of walk.cuh in WALK_VOTE mode.
// ------------------------------------------------------------------------------------------------
int hough_vote_tiled(hough_plan* p, const float* d_hits_xy, int32_t n_hits, const int32_t* d_event_offsets,
                     int32_t n_events, void* d_accum, cudaStream_t st) {
    if (p->tile_max_cols < 1) return hough_vote_fullscan(p, d_hits_xy, n_hits, d_event_offsets, n_events, d_accum, st);
    const int rc = hough_stage_hits(p, d_hits_xy, n_hits, d_event_offsets, n_events, st, false);
    if (rc != HOUGH_OK) return rc;
    WalkArgs a{};
    a.staged = p->d_staged;
    a.off = d_event_offsets;
    a.key_start = p->d_stage_cnt;
    walk_shape(p, n_events, a.n_slabs, a.slab_cols);
    a.stride = p->tile_stride_words;
    a.accum = d_accum;
    return walk_dispatch<WALK_VOTE>(p, n_events, a, p->tile32 != 0, p->c.is_u16 != 0, st);
}

extern "C" int hough_vote(hough_plan* p, const float* d_hits_xy, int32_t n_hits, const int32_t* d_event_offsets,
                          int32_t n_events, void* d_accum, void* cuda_stream) {
    if (!p || !d_event_offsets || !d_accum) return HOUGH_ERR_INVALID_ARG;
    if (n_hits < 0 || n_events < 0 || n_hits > p->max_hits || n_events > p->max_events) return HOUGH_ERR_INVALID_ARG;
    if (n_hits > 0 && !d_hits_xy) return HOUGH_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(d_hits_xy) & 7u) || (reinterpret_cast<uintptr_t>(d_accum) & 3u))
        return HOUGH_ERR_INVALID_ARG;
    if (n_events == 0) return n_hits == 0 ? HOUGH_OK : HOUGH_ERR_INVALID_ARG;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    if (p->fullscan) return hough_vote_fullscan(p, d_hits_xy, n_hits, d_event_offsets, n_events, d_accum, st);
    return hough_vote_tiled(p, d_hits_xy, n_hits, d_event_offsets, n_events, d_accum, st);
}

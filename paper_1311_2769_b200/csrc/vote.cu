// vote.cu -- A1/A2/A3: hit staging, vote, flush (D3/D4).
#include "common.cuh"

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
        const int j = d3_bin_from_w(w, r2, d.x, d.y, d.z, c.A_f, c.qmin, c.inv_wq, c.nq_f);
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
// Tiled path (A2/A3).  One CTA owns the tile (event e, d0 slice k, phi0 columns [c0, c0 + cols)) of the
// accumulator in shared memory (two 16-bit bins per word, or 32-bit bins), so no vote ever needs a global
// atomic and the tile is written to HBM exactly once, which also implements "overwrite" (S8).
//
// Work mapping: lane = hit.  A warp takes 32 consecutive staged hits of one radius class (same window length,
// neighbouring azimuth thanks to the (class, sector) sort of stage.cu); every lane walks the `steps` columns of
// its own window, evaluating the exact D3 sequence at each and adding its vote with a shared-memory atomic.
// Lanes stay converged because `steps` is a property of (class, k); lane efficiency does not depend on the
// window length (2 columns on the innermost layer, 220 on the outermost at n_phi = 1024).
// ------------------------------------------------------------------------------------------------
namespace {

constexpr int VOTE_THREADS = 256;
constexpr int VOTE_WARPS = VOTE_THREADS / 32;

struct VoteSmem {
    uint32_t* tile;      // [cols * stride]
    float2* cs;          // [cols]
    float* lo;           // [n_class]
    int* steps;          // [n_class]
    int* seg_start;      // [2 * n_class]   first staged hit (relative to the event) of each segment
    int* seg_cnt;        // [2 * n_class]
    int* seg_pref;       // [2 * n_class + 1] exclusive prefix of 32-hit batches
};

__host__ __device__ inline size_t vote_smem_bytes(int cols, int stride, int n_class) {
    size_t b = ((size_t)cols * stride * 4 + 15) & ~(size_t)15;
    b += (size_t)cols * 8;
    b += (size_t)n_class * 8;
    b += (size_t)n_class * 2 * 8 + ((size_t)n_class * 2 + 1) * 4;
    return (b + 15) & ~(size_t)15;
}

template <bool TILE32, bool OUT16, bool FULLPHI>
__global__ void __launch_bounds__(VOTE_THREADS, 3)
vote_tiled_kernel(HoughConsts c, const float4* __restrict__ staged, const int32_t* __restrict__ off,
                  const int32_t* __restrict__ key_start, void* __restrict__ accum, int n_slabs, int slab_cols,
                  int stride) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int slab = blockIdx.x % n_slabs;
    const int k = (blockIdx.x / n_slabs) % c.n_d0;
    const int e = blockIdx.x / (n_slabs * c.n_d0);
    const int c0 = slab * slab_cols;
    const int cols = min(slab_cols, c.n_phi - c0);
    const int nphi = c.n_phi;
    const int nc = c.n_class;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    VoteSmem s;
    {
        unsigned char* q = smem_raw;
        s.tile = reinterpret_cast<uint32_t*>(q);  q += ((size_t)slab_cols * stride * 4 + 15) & ~(size_t)15;
        s.cs = reinterpret_cast<float2*>(q);      q += (size_t)slab_cols * 8;
        s.lo = reinterpret_cast<float*>(q);       q += (size_t)nc * 4;
        s.steps = reinterpret_cast<int*>(q);      q += (size_t)nc * 4;
        s.seg_start = reinterpret_cast<int*>(q);  q += (size_t)nc * 2 * 4;
        s.seg_cnt = reinterpret_cast<int*>(q);    q += (size_t)nc * 2 * 4;
        s.seg_pref = reinterpret_cast<int*>(q);
    }

    // ---- prologue: zero the tile, load tables, list the segments of staged hits that can reach the tile ----
    {
        uint4* t4 = reinterpret_cast<uint4*>(s.tile);
        const int n4 = (cols * stride + 3) >> 2;
        for (int x = tid; x < n4; x += VOTE_THREADS) t4[x] = make_uint4(0u, 0u, 0u, 0u);
        for (int x = tid; x < cols; x += VOTE_THREADS) s.cs[x] = __ldg(c.cs + c0 + x);
    }
    const int ev_begin = __ldg(off + e);
    const int32_t* ks = key_start + (size_t)e * (c.n_keys + 1);
    for (int cl = tid; cl < nc; cl += VOTE_THREADS) {
        const int2 w = __ldg(c.win + (size_t)cl * c.n_d0 + k);
        const float lo = __int_as_float(w.x);
        const int steps = w.y;
        s.lo[cl] = lo;
        s.steps[cl] = steps;
        int a0 = 0, n0 = 0, a1 = 0, n1 = 0;
        if (steps > 0) {
            const int NS = c.n_sector;
            int sa = 0, ns = NS;
            if (!FULLPHI) {
                // hits whose window [ceil(u + lo), +steps) meets [c0, c0 + cols): u in (c0 - steps - lo, c0 + cols - lo)
                const float W = (float)nphi / (float)NS;
                const float ua = (float)(c0 - steps) - lo - 2.0f;
                const float ub = (float)(c0 + cols) - lo + 2.0f;
                const int s0 = (int)floorf((ua + 0.5f) / W);
                const int s1 = (int)floorf((ub + 0.5f) / W);
                ns = s1 - s0 + 1;
                if (ns >= NS) { sa = 0; ns = NS; }
                else { sa = s0 % NS; if (sa < 0) sa += NS; }
            }
            const int base = cl * NS;
            if (sa + ns <= NS) {
                a0 = __ldg(ks + base + sa);
                n0 = __ldg(ks + base + sa + ns) - a0;
            } else {
                a0 = __ldg(ks + base + sa);
                n0 = __ldg(ks + base + NS) - a0;
                a1 = __ldg(ks + base);
                n1 = __ldg(ks + base + (sa + ns - NS)) - a1;
            }
        }
        s.seg_start[2 * cl] = a0;     s.seg_cnt[2 * cl] = n0;
        s.seg_start[2 * cl + 1] = a1; s.seg_cnt[2 * cl + 1] = n1;
    }
    __syncthreads();
    if (warp == 0) {                                    // exclusive prefix of batch counts over 2*nc segments
        const int nseg = 2 * nc;
        const int per = (nseg + 31) / 32;
        int sum = 0;
        for (int x = lane * per; x < min(nseg, (lane + 1) * per); ++x) sum += (s.seg_cnt[x] + 31) >> 5;
        int incl = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += y;
        }
        int run = incl - sum;
        for (int x = lane * per; x < min(nseg, (lane + 1) * per); ++x) {
            s.seg_pref[x] = run;
            run += (s.seg_cnt[x] + 31) >> 5;
        }
        if (lane == 31) s.seg_pref[nseg] = incl;
    }
    __syncthreads();

    // ---- main loop: 32-hit batches, static round-robin over the CTA's warps ----
    const int n_batches = s.seg_pref[2 * nc];
    const float4 d = __ldg(c.d0t + k);
    for (int bt = warp; bt < n_batches; bt += VOTE_WARPS) {
        int lo_i = 0, hi_i = 2 * nc;                    // largest segment with seg_pref[seg] <= bt
        while (hi_i - lo_i > 1) {
            const int mid = (lo_i + hi_i) >> 1;
            if (s.seg_pref[mid] <= bt) lo_i = mid; else hi_i = mid;
        }
        const int seg = lo_i;
        const int in_seg = (bt - s.seg_pref[seg]) * 32 + lane;
        const bool active = in_seg < s.seg_cnt[seg];
        const int cl = seg >> 1;
        const int steps = s.steps[cl];
        float4 hv = make_float4(0.f, 0.f, 0.f, 0.f);
        if (active) hv = __ldg(staged + ev_begin + s.seg_start[seg] + in_seg);
        const float x = hv.x, y = hv.y;
        const float r2 = d3_r2(x, y);
        int i_lo = (int)ceilf(hv.z + s.lo[cl]);
        if (i_lo < 0) i_lo += nphi;
        if (i_lo >= nphi) i_lo -= nphi;
        if (!(i_lo >= 0 && i_lo < nphi)) i_lo = 0;
        int col, t_cnt;
        if (FULLPHI) {
            col = i_lo;
            t_cnt = steps;
        } else {
            int dd = i_lo - c0;                          // column relative to the tile, cyclic
            if (dd < 0) dd += nphi;
            const bool inside = dd < cols;
            int t_begin = inside ? 0 : nphi - dd;
            int t_end = inside ? min(steps, cols - dd) : min(steps, nphi - dd + cols);
            if (steps + cols > nphi) { t_begin = 0; t_end = steps; }       // a window could re-enter the tile
            if (!active || t_begin >= t_end) { t_begin = 0x7fffffff; t_end = 0; }
            const int tb = __reduce_min_sync(0xffffffffu, t_begin);
            const int te = __reduce_max_sync(0xffffffffu, t_end);
            if (tb >= te) continue;
            col = dd + tb;
            if (col >= nphi) col -= nphi;
            t_cnt = te - tb;
        }
#pragma unroll 2
        for (int t = 0; t < t_cnt; ++t) {
            const bool in_tile = FULLPHI ? true : (col < cols);
            const float2 cs = s.cs[in_tile ? col : 0];
            float w, f;
            d3_wf(x, y, cs.x, cs.y, w, f);
            const int j = d3_bin_from_w(w, r2, d.x, d.y, d.z, c.A_f, c.qmin, c.inv_wq, c.nq_f);
            if (active && in_tile && f > 0.0f && j >= 0) {
                if (TILE32) atomicAdd(s.tile + col * stride + j, 1u);
                else atomicAdd(s.tile + col * stride + (j >> 1), (j & 1) ? 0x10000u : 1u);
            }
            ++col;
            if (col == nphi) col = 0;
        }
    }
    __syncthreads();

    // ---- flush: the tile is written to the global accumulator exactly once (A3) ----
    const int nq = c.n_qpt;
    const size_t row0 = ((size_t)e * c.n_d0 + k) * (size_t)nphi + c0;      // first global row of the tile
    if (TILE32) {
        int* g = reinterpret_cast<int*>(accum) + row0 * nq;
        for (int ci = warp; ci < cols; ci += VOTE_WARPS)
            for (int j = lane; j < nq; j += 32) g[(size_t)ci * nq + j] = (int)s.tile[ci * stride + j];
    } else if (OUT16) {
        if ((nq & 1) == 0) {
            uint32_t* g = reinterpret_cast<uint32_t*>(reinterpret_cast<unsigned short*>(accum) + row0 * nq);
            const int rw = nq >> 1;
            for (int ci = warp; ci < cols; ci += VOTE_WARPS)
                for (int jw = lane; jw < rw; jw += 32) g[(size_t)ci * rw + jw] = s.tile[ci * stride + jw];
        } else {
            unsigned short* g = reinterpret_cast<unsigned short*>(accum) + row0 * nq;
            for (int ci = warp; ci < cols; ci += VOTE_WARPS)
                for (int j = lane; j < nq; j += 32)
                    g[(size_t)ci * nq + j] = (unsigned short)((s.tile[ci * stride + (j >> 1)] >> (16 * (j & 1))) & 0xffffu);
        }
    } else {
        int* g = reinterpret_cast<int*>(accum) + row0 * nq;
        if ((nq & 1) == 0) {
            const int rw = nq >> 1;
            for (int ci = warp; ci < cols; ci += VOTE_WARPS)
                for (int jw = lane; jw < rw; jw += 32) {
                    const uint32_t v = s.tile[ci * stride + jw];
                    *reinterpret_cast<int2*>(g + (size_t)ci * nq + 2 * jw) = make_int2((int)(v & 0xffffu), (int)(v >> 16));
                }
        } else {
            for (int ci = warp; ci < cols; ci += VOTE_WARPS)
                for (int j = lane; j < nq; j += 32)
                    g[(size_t)ci * nq + j] = (int)((s.tile[ci * stride + (j >> 1)] >> (16 * (j & 1))) & 0xffffu);
        }
    }
}

template <bool TILE32, bool OUT16, bool FULLPHI>
int launch_vote_tiled(hough_plan* p, int n_events, void* d_accum, int n_slabs, int slab_cols, cudaStream_t st) {
    const size_t smem = vote_smem_bytes(slab_cols, p->tile_stride_words, p->c.n_class);
    auto kern = vote_tiled_kernel<TILE32, OUT16, FULLPHI>;
    HOUGH_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const long long grid = (long long)n_slabs * p->c.n_d0 * n_events;
    if (grid > 0x7fffffffLL) return HOUGH_ERR_UNSUPPORTED;
    kern<<<(unsigned)grid, VOTE_THREADS, smem, st>>>(p->c, p->d_staged, p->vote_offsets, p->d_stage_cnt, d_accum, n_slabs,
                                                     slab_cols, p->tile_stride_words);
    HOUGH_CUDA_TRY(cudaGetLastError());
    hough_count_launches(1);
    return HOUGH_OK;
}

}  // namespace

int hough_vote_tiled(hough_plan* p, const float* d_hits_xy, int32_t n_hits, const int32_t* d_event_offsets,
                     int32_t n_events, void* d_accum, cudaStream_t st) {
    if (p->tile_max_cols < 1) return hough_vote_fullscan(p, d_hits_xy, n_hits, d_event_offsets, n_events, d_accum, st);
    int rc = hough_stage_hits(p, d_hits_xy, n_hits, d_event_offsets, n_events, st);
    if (rc != HOUGH_OK) return rc;
    // tile shape: as many columns as fit the shared-memory budget, then split further until the grid fills the GPU
    const int nphi = p->c.n_phi;
    int n_slabs = (nphi + p->tile_max_cols - 1) / p->tile_max_cols;
    const long long want = 3LL * p->sm_count;
    while ((long long)n_slabs * p->c.n_d0 * n_events < want && (nphi + n_slabs - 1) / n_slabs > 32) n_slabs *= 2;
    const int slab_cols = (nphi + n_slabs - 1) / n_slabs;
    n_slabs = (nphi + slab_cols - 1) / slab_cols;
    p->vote_offsets = d_event_offsets;
    const bool out16 = p->c.is_u16 != 0;
    const bool full = n_slabs == 1;
    if (p->tile32) {
        return full ? launch_vote_tiled<true, false, true>(p, n_events, d_accum, n_slabs, slab_cols, st)
                    : launch_vote_tiled<true, false, false>(p, n_events, d_accum, n_slabs, slab_cols, st);
    }
    if (out16) {
        return full ? launch_vote_tiled<false, true, true>(p, n_events, d_accum, n_slabs, slab_cols, st)
                    : launch_vote_tiled<false, true, false>(p, n_events, d_accum, n_slabs, slab_cols, st);
    }
    return full ? launch_vote_tiled<false, false, true>(p, n_events, d_accum, n_slabs, slab_cols, st)
                : launch_vote_tiled<false, false, false>(p, n_events, d_accum, n_slabs, slab_cols, st);
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

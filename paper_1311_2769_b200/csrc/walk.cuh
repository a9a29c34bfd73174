// walk.cuh -- the column walk shared by the vote (A2/A3, vote.cu) and the hit association (A5, assign.cu).
//
// One CTA owns the tile (event e, d0 slice k, phi0 columns [c0, c0 + cols)) in shared memory:
//   WALK_VOTE   : the tile is that part of the accumulator (two 16-bit bins per word, or 32-bit bins); votes
//                 are shared-memory atomics, the tile is written to HBM exactly once (no global atomic; this
//                 also implements "overwrite", S8).
//   WALK_ASSIGN : the tile holds votes + 1 at the bins of the event's candidates (0 elsewhere), scattered
//                 from the candidate list; every vote position of a hit probes bins jh - dj .. jh + dj and
//                 keeps the best D8 key; one atomicMax per (hit, tile) publishes it.
//
// Work mapping: lane = hit.  A warp takes 32 consecutive staged hits of one radius class (same window length,
// neighbouring azimuth thanks to the (class, sector) sort of stage.cu); every lane walks the `steps` columns of
// its own window and evaluates the exact D3 sequence at each.  Lanes stay converged because `steps` is a
// property of (class, k); lane efficiency does not depend on the window length (2 columns on the innermost
// layer, 220 on the outermost at n_phi = 1024).
#pragma once

#include "common.cuh"

constexpr int WALK_VOTE = 0;
constexpr int WALK_ASSIGN = 1;
constexpr int WALK_THREADS = 256;
constexpr int WALK_WARPS = WALK_THREADS / 32;

struct WalkArgs {
    const float4* staged;            // [n_hits] staged hits (stage.cu)
    const int32_t* off;              // [n_events + 1] event offsets
    const int32_t* key_start;        // [n_events][n_keys + 1] exclusive key starts
    int n_slabs, slab_cols, stride;  // tile shape
    // WALK_VOTE
    void* accum;
    // WALK_ASSIGN
    const hough_candidate* cands;
    const int2* slice;               // [n_events * n_d0 * n_slabs] {first, end} candidate of each tile
    int assoc_dj;
    unsigned long long* best_key;    // [n_hits] by original hit index
};

__host__ __device__ inline size_t walk_smem_bytes(int cols, int stride, int n_class) {
    size_t b = ((size_t)cols * stride * 4 + 15) & ~(size_t)15;
    b += (size_t)cols * 8;                                              // cos/sin of the tile's columns
    b += (size_t)n_class * 8;                                           // lo_off, steps
    b += (size_t)n_class * 2 * 8 + ((size_t)n_class * 2 + 1) * 4;       // segments
    return (b + 15) & ~(size_t)15;
}

// D8 key with the candidate's linear bin in place of its index: inside one event the candidate list is sorted
// by linear bin (D6), so both orders agree.
__device__ __forceinline__ unsigned long long walk_key(unsigned votes, int adj, unsigned linbin) {
    return ((unsigned long long)votes << 40) | ((unsigned long long)(255 - adj) << 32) |
           (unsigned long long)(0xFFFFFFFFu - linbin);
}

// votes of the candidate at (i, j) among cands[first, end) (one event, one d0 slice: sorted by (i, j))
static __device__ __noinline__ unsigned walk_lookup_votes(const hough_candidate* __restrict__ cands, int first, int end, int i, int j) {
    int lo = first, hi = end;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        const int4 q = __ldg(reinterpret_cast<const int4*>(cands + mid));
        if (q.z < i || (q.z == i && q.w < j)) lo = mid + 1; else hi = mid;
    }
    return lo < end ? (unsigned)__ldg(&cands[lo].votes) : 0u;
}

template <int MODE, bool TILE32, bool OUT16, bool FULLPHI>
__global__ void __launch_bounds__(WALK_THREADS, 3) walk_kernel(HoughConsts c, WalkArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n_slabs = a.n_slabs, slab_cols = a.slab_cols, stride = a.stride;
    const int slab = blockIdx.x % n_slabs;
    const int k = (blockIdx.x / n_slabs) % c.n_d0;
    const int e = blockIdx.x / (n_slabs * c.n_d0);
    const int c0 = slab * slab_cols;
    const int cols = min(slab_cols, c.n_phi - c0);
    const int nphi = c.n_phi;
    const int nq = c.n_qpt;
    const int nc = c.n_class;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    uint32_t* s_tile; float2* s_cs; float* s_lo; int* s_steps; int* s_seg_start; int* s_seg_cnt; int* s_seg_pref;
    {
        unsigned char* q = smem_raw;
        s_tile = reinterpret_cast<uint32_t*>(q);  q += ((size_t)slab_cols * stride * 4 + 15) & ~(size_t)15;
        s_cs = reinterpret_cast<float2*>(q);      q += (size_t)slab_cols * 8;
        s_lo = reinterpret_cast<float*>(q);       q += (size_t)nc * 4;
        s_steps = reinterpret_cast<int*>(q);      q += (size_t)nc * 4;
        s_seg_start = reinterpret_cast<int*>(q);  q += (size_t)nc * 2 * 4;
        s_seg_cnt = reinterpret_cast<int*>(q);    q += (size_t)nc * 2 * 4;
        s_seg_pref = reinterpret_cast<int*>(q);
    }

    int cand_first = 0, cand_end = 0;
    if (MODE == WALK_ASSIGN) {
        const int2 sl = __ldg(a.slice + blockIdx.x);
        cand_first = sl.x; cand_end = sl.y;
        if (cand_first >= cand_end) return;              // no candidate in this tile: nothing to associate
    }

    // ---- prologue: zero the tile, load tables, list the segments of staged hits that can reach the tile ----
    {
        uint4* t4 = reinterpret_cast<uint4*>(s_tile);
        const int n4 = (cols * stride + 3) >> 2;
        for (int x = tid; x < n4; x += WALK_THREADS) t4[x] = make_uint4(0u, 0u, 0u, 0u);
        for (int x = tid; x < cols; x += WALK_THREADS) s_cs[x] = __ldg(c.cs + c0 + x);
    }
    const int ev_begin = __ldg(a.off + e);
    const int32_t* ks = a.key_start + (size_t)e * (c.n_keys + 1);
    for (int cl = tid; cl < nc; cl += WALK_THREADS) {
        const int2 w = __ldg(c.win + (size_t)cl * c.n_d0 + k);
        const float lo = __int_as_float(w.x);
        const int steps = w.y;
        s_lo[cl] = lo;
        s_steps[cl] = steps;
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
        s_seg_start[2 * cl] = a0;     s_seg_cnt[2 * cl] = n0;
        s_seg_start[2 * cl + 1] = a1; s_seg_cnt[2 * cl + 1] = n1;
    }
    __syncthreads();
    if (warp == 0) {                                    // exclusive prefix of batch counts over 2*nc segments
        const int nseg = 2 * nc;
        const int per = (nseg + 31) / 32;
        int sum = 0;
        for (int x = lane * per; x < min(nseg, (lane + 1) * per); ++x) sum += (s_seg_cnt[x] + 31) >> 5;
        int incl = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += y;
        }
        int run = incl - sum;
        for (int x = lane * per; x < min(nseg, (lane + 1) * per); ++x) {
            s_seg_pref[x] = run;
            run += (s_seg_cnt[x] + 31) >> 5;
        }
        if (lane == 31) s_seg_pref[nseg] = incl;
    }
    if (MODE == WALK_ASSIGN) {                          // scatter votes + 1 of this tile's candidates
        for (int ci = cand_first + tid; ci < cand_end; ci += WALK_THREADS) {
            const int4 q = __ldg(reinterpret_cast<const int4*>(a.cands + ci));          // event, k, i, j
            const unsigned v = (unsigned)__ldg(&a.cands[ci].votes) + 1u;
            const int col = q.z - c0;
            if (TILE32) s_tile[col * stride + q.w] = v;
            else reinterpret_cast<unsigned short*>(s_tile)[col * stride * 2 + q.w] = (unsigned short)min(v, 65535u);
        }
    }
    __syncthreads();

    // ---- main loop: 32-hit batches, static round-robin over the CTA's warps ----
    const int n_batches = s_seg_pref[2 * nc];
    const float4 d = __ldg(c.d0t + k);
    const unsigned row_lin0 = (unsigned)(k * nphi + c0) * (unsigned)nq;   // linear bin of (k, c0, 0) inside the event
    for (int bt = warp; bt < n_batches; bt += WALK_WARPS) {
        int lo_i = 0, hi_i = 2 * nc;                    // largest segment with seg_pref[seg] <= bt
        while (hi_i - lo_i > 1) {
            const int mid = (lo_i + hi_i) >> 1;
            if (s_seg_pref[mid] <= bt) lo_i = mid; else hi_i = mid;
        }
        const int seg = lo_i;
        const int in_seg = (bt - s_seg_pref[seg]) * 32 + lane;
        const bool active = in_seg < s_seg_cnt[seg];
        const int cl = seg >> 1;
        const int steps = s_steps[cl];
        float4 hv = make_float4(0.f, 0.f, 0.f, 0.f);
        if (active) hv = __ldg(a.staged + ev_begin + s_seg_start[seg] + in_seg);
        const float x = hv.x, y = hv.y;
        const float r2 = d3_r2(x, y);
        int i_lo = (int)ceilf(hv.z + s_lo[cl]);
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
        unsigned long long best = 0ull;
#pragma unroll 2
        for (int t = 0; t < t_cnt; ++t) {
            const bool in_tile = FULLPHI ? true : (col < cols);
            const float2 cs = s_cs[in_tile ? col : 0];
            float w, f;
            d3_wf(x, y, cs.x, cs.y, w, f);
            const int j = d3_bin_from_w(w, r2, d.x, d.y, d.z, c.A_f, c.qmin, c.inv_wq, c.nq_f);
            if (active && in_tile && f > 0.0f && j >= 0) {
                if (MODE == WALK_VOTE) {
                    if (TILE32) atomicAdd(s_tile + col * stride + j, 1u);
                    else atomicAdd(s_tile + col * stride + (j >> 1), (j & 1) ? 0x10000u : 1u);
                } else {
                    const int j0 = max(j - a.assoc_dj, 0), j1 = min(j + a.assoc_dj, nq - 1);
                    for (int jj = j0; jj <= j1; ++jj) {
                        unsigned v;
                        if (TILE32) v = s_tile[col * stride + jj];
                        else v = reinterpret_cast<const unsigned short*>(s_tile)[col * stride * 2 + jj];
                        if (v) {
                            if (!TILE32 && v == 65535u)      // saturated 16-bit entry: take the votes from the record
                                v = walk_lookup_votes(a.cands, cand_first, cand_end, c0 + col, jj) + 1u;
                            const unsigned long long key = walk_key(v - 1u, abs(jj - j), row_lin0 + (unsigned)(col * nq + jj));
                            best = key > best ? key : best;
                        }
                    }
                }
            }
            ++col;
            if (col == nphi) col = 0;
        }
        if (MODE == WALK_ASSIGN) {
            if (best) atomicMax(a.best_key + __float_as_int(hv.w), best);
        }
    }
    if (MODE == WALK_ASSIGN) return;
    __syncthreads();

    // ---- flush: the tile is written to the global accumulator exactly once (A3) ----
    const size_t row0 = ((size_t)e * c.n_d0 + k) * (size_t)nphi + c0;      // first global row of the tile
    if (TILE32) {
        int* g = reinterpret_cast<int*>(a.accum) + row0 * nq;
        for (int ci = warp; ci < cols; ci += WALK_WARPS)
            for (int j = lane; j < nq; j += 32) g[(size_t)ci * nq + j] = (int)s_tile[ci * stride + j];
    } else if (OUT16) {
        if ((nq & 1) == 0) {
            uint32_t* g = reinterpret_cast<uint32_t*>(reinterpret_cast<unsigned short*>(a.accum) + row0 * nq);
            const int rw = nq >> 1;
            for (int ci = warp; ci < cols; ci += WALK_WARPS)
                for (int jw = lane; jw < rw; jw += 32) g[(size_t)ci * rw + jw] = s_tile[ci * stride + jw];
        } else {
            unsigned short* g = reinterpret_cast<unsigned short*>(a.accum) + row0 * nq;
            for (int ci = warp; ci < cols; ci += WALK_WARPS)
                for (int j = lane; j < nq; j += 32)
                    g[(size_t)ci * nq + j] = (unsigned short)((s_tile[ci * stride + (j >> 1)] >> (16 * (j & 1))) & 0xffffu);
        }
    } else {
        int* g = reinterpret_cast<int*>(a.accum) + row0 * nq;
        if ((nq & 1) == 0) {
            const int rw = nq >> 1;
            for (int ci = warp; ci < cols; ci += WALK_WARPS)
                for (int jw = lane; jw < rw; jw += 32) {
                    const uint32_t v = s_tile[ci * stride + jw];
                    *reinterpret_cast<int2*>(g + (size_t)ci * nq + 2 * jw) = make_int2((int)(v & 0xffffu), (int)(v >> 16));
                }
        } else {
            for (int ci = warp; ci < cols; ci += WALK_WARPS)
                for (int j = lane; j < nq; j += 32)
                    g[(size_t)ci * nq + j] = (int)((s_tile[ci * stride + (j >> 1)] >> (16 * (j & 1))) & 0xffffu);
        }
    }
}

// tile shape of a call: as many columns as fit the shared-memory budget, then split further until the grid
// fills the GPU
inline void walk_shape(const hough_plan* p, int n_events, int& n_slabs, int& slab_cols) {
    const int nphi = p->c.n_phi;
    n_slabs = (nphi + p->tile_max_cols - 1) / p->tile_max_cols;
    const long long want = 3LL * p->sm_count;
    while ((long long)n_slabs * p->c.n_d0 * n_events < want && (nphi + n_slabs - 1) / n_slabs > 32) n_slabs *= 2;
    slab_cols = (nphi + n_slabs - 1) / n_slabs;
    n_slabs = (nphi + slab_cols - 1) / slab_cols;
}

template <int MODE, bool TILE32, bool OUT16, bool FULLPHI>
int walk_launch(hough_plan* p, int n_events, WalkArgs a, cudaStream_t st) {
    const size_t smem = walk_smem_bytes(a.slab_cols, a.stride, p->c.n_class);
    auto kern = walk_kernel<MODE, TILE32, OUT16, FULLPHI>;
    static size_t smem_configured = 0;              // per instantiation; raised only when a call needs more
    if (smem > smem_configured) {
        HOUGH_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        smem_configured = smem;
    }
    const long long grid = (long long)a.n_slabs * p->c.n_d0 * n_events;
    if (grid > 0x7fffffffLL) return HOUGH_ERR_UNSUPPORTED;
    kern<<<(unsigned)grid, WALK_THREADS, smem, st>>>(p->c, a);
    HOUGH_CUDA_TRY(cudaGetLastError());
    hough_count_launches(1);
    return HOUGH_OK;
}

template <int MODE>
int walk_dispatch(hough_plan* p, int n_events, WalkArgs a, bool tile32, bool out16, cudaStream_t st) {
    const bool full = a.n_slabs == 1;
    if (tile32)
        return full ? walk_launch<MODE, true, false, true>(p, n_events, a, st)
                    : walk_launch<MODE, true, false, false>(p, n_events, a, st);
    if (out16 && MODE == WALK_VOTE)
        return full ? walk_launch<MODE, false, true, true>(p, n_events, a, st)
                    : walk_launch<MODE, false, true, false>(p, n_events, a, st);
    return full ? walk_launch<MODE, false, false, true>(p, n_events, a, st)
                : walk_launch<MODE, false, false, false>(p, n_events, a, st);
}

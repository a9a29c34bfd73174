// assign.cu -- A5: hit-to-candidate association and duplicate removal (D8/D9).
//
// Tiled path (default):
//   K1       : stage the hits (stage.cu), exactly as for the vote
//   K4-slice : candidate range of every (event, d0 slice, phi0 slab) tile by binary search in the sorted list
//   K4a      : the column walk of walk.cuh in WALK_ASSIGN mode -> 64-bit best key per hit (atomicMax)
//   K4b      : decode best key (linear bin) -> candidate index by binary search; count hits per candidate
//   K4c      : keep = nhits >= min_hits; hits of dropped candidates -> -1
// Full-scan path (plan option "fullscan", or rows too long for a tile): a bitmask + rank index over all bins
// and one thread per (hit, phi0 column), no windowing.
#include "walk.cuh"

namespace {

__device__ __forceinline__ int find_event_a(const int32_t* __restrict__ off, int n_events, int h) {
    int lo = 0, hi = n_events;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (off[mid] <= h) lo = mid; else hi = mid;
    }
    return lo;
}

__global__ void __launch_bounds__(256) cand_index_kernel(HoughConsts c, const hough_candidate* __restrict__ cands,
                                                         const int32_t* __restrict__ cand_offsets, int n_events,
                                                         int capacity, uint32_t* __restrict__ mask,
                                                         int32_t* __restrict__ word_rank) {
    const int total = min(cand_offsets[n_events], capacity);
    for (int ci = blockIdx.x * blockDim.x + threadIdx.x; ci < total; ci += gridDim.x * blockDim.x) {
        const int4 a = __ldg(reinterpret_cast<const int4*>(cands + ci));        // event, k, i, j
        const int b = (a.y * c.n_phi + a.z) * c.n_qpt + a.w;
        const size_t word = (size_t)a.x * c.words_per_event + (b >> 5);
        atomicOr(mask + word, 1u << (b & 31));
        bool first = ci == 0;
        if (!first) {
            const int4 q = __ldg(reinterpret_cast<const int4*>(cands + ci - 1));
            const int bq = (q.y * c.n_phi + q.z) * c.n_qpt + q.w;
            first = q.x != a.x || (bq >> 5) != (b >> 5);
        }
        if (first) word_rank[word] = ci;
    }
}

__device__ __forceinline__ unsigned long long make_key(int votes, int adj, int index) {
    return ((unsigned long long)(unsigned)votes << 40) | ((unsigned long long)(255 - adj) << 32) |
           (unsigned long long)(0xFFFFFFFFu - (unsigned)index);
}

// full-scan association: one thread per (hit, phi0 column)
__global__ void __launch_bounds__(256) assign_fullscan_kernel(HoughConsts c, const float2* __restrict__ hits, int n_hits,
                                                              const int32_t* __restrict__ off, int n_events,
                                                              const hough_candidate* __restrict__ cands,
                                                              const uint32_t* __restrict__ mask,
                                                              const int32_t* __restrict__ word_rank, int assoc_dj,
                                                              const uint8_t* __restrict__ keep,
                                                              unsigned long long* __restrict__ best_key) {
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
    const int e = find_event_a(off, n_events, h);
    const uint32_t* emask = mask + (size_t)e * c.words_per_event;
    const int32_t* erank = word_rank + (size_t)e * c.words_per_event;
    unsigned long long best = 0ull;
    for (int k = 0; k < c.n_d0; ++k) {
        const float4 d = c.d0t[k];
        const int jh = d3_bin_from_w(w, r2, d.x, d.y, d.z, c.A_f, c.qmin, c.inv_wq, c.nq_f, c.model != 0);
        if (jh < 0) continue;
        const int row = (k * c.n_phi + i) * c.n_qpt;
        const int j0 = max(jh - assoc_dj, 0), j1 = min(jh + assoc_dj, c.n_qpt - 1);
        for (int j = j0; j <= j1; ++j) {
            const int b = row + j;
            const uint32_t m = __ldg(emask + (b >> 5));
            if (!((m >> (b & 31)) & 1u)) continue;
            const int ci = __ldg(erank + (b >> 5)) + __popc(m & ((1u << (b & 31)) - 1u));
            if (keep && !__ldg(keep + ci)) continue;
            const int votes = __ldg(&cands[ci].votes);
            const unsigned long long key = make_key(votes, abs(jh - j), ci);
            best = key > best ? key : best;
        }
    }
    if (best) atomicMax(best_key + h, best);
}

__global__ void __launch_bounds__(256) assign_decode_kernel(const unsigned long long* __restrict__ best_key, int n_hits,
                                                            int32_t* __restrict__ hit_to_cand,
                                                            int32_t* __restrict__ cand_nhits) {
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= n_hits) return;
    const unsigned long long key = best_key[h];
    int ci = -1;
    if (key) {
        ci = (int)(0xFFFFFFFFu - (unsigned)(key & 0xFFFFFFFFull));
        atomicAdd(cand_nhits + ci, 1);
    }
    hit_to_cand[h] = ci;
}

// {first, end} candidate of tile (event e, slice k, slab): lower bounds of the tile's first and last+1 linear
// bins among the event's participating candidates (rank < capacity)
__global__ void __launch_bounds__(256) cand_slice_kernel(HoughConsts c, const hough_candidate* __restrict__ cands,
                                                         const int32_t* __restrict__ cand_offsets, int n_events,
                                                         int capacity, int n_slabs, int slab_cols,
                                                         int2* __restrict__ slice) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_events * c.n_d0 * n_slabs) return;
    const int slab = t % n_slabs;
    const int k = (t / n_slabs) % c.n_d0;
    const int e = t / (n_slabs * c.n_d0);
    const int first = min(__ldg(cand_offsets + e), capacity), end = min(__ldg(cand_offsets + e + 1), capacity);
    const int c0 = slab * slab_cols, c1 = min(c0 + slab_cols, c.n_phi);
    int2 out;
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        const int ti = s ? c1 : c0;                 // lower bound of (k, ti, 0); (k, n_phi, 0) == (k + 1, 0, 0)
        int lo = first, hi = end;
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            const int4 q = __ldg(reinterpret_cast<const int4*>(cands + mid));    // event, k, i, j
            if (q.y < k || (q.y == k && q.z < ti)) lo = mid + 1; else hi = mid;
        }
        if (s) out.y = lo; else out.x = lo;
    }
    slice[t] = out;
}

// best key -> candidate index: the key's low word is ~(linear bin); the event's candidates are sorted by it
__global__ void __launch_bounds__(256) assign_decode_bin_kernel(HoughConsts c, const unsigned long long* __restrict__ best_key,
                                                                int n_hits, const int32_t* __restrict__ off, int n_events,
                                                                const hough_candidate* __restrict__ cands,
                                                                const int32_t* __restrict__ cand_offsets, int capacity,
                                                                int32_t* __restrict__ hit_to_cand,
                                                                int32_t* __restrict__ cand_nhits) {
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= n_hits) return;
    const unsigned long long key = best_key[h];
    int ci = -1;
    if (key) {
        const unsigned lin = 0xFFFFFFFFu - (unsigned)(key & 0xFFFFFFFFull);
        const int e = find_event_a(off, n_events, h);
        int lo = min(__ldg(cand_offsets + e), capacity), hi = min(__ldg(cand_offsets + e + 1), capacity);
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            const int4 q = __ldg(reinterpret_cast<const int4*>(cands + mid));
            const unsigned lm = (unsigned)(q.y * c.n_phi + q.z) * (unsigned)c.n_qpt + (unsigned)q.w;
            if (lm < lin) lo = mid + 1; else hi = mid;
        }
        ci = lo;
        atomicAdd(cand_nhits + ci, 1);
    }
    hit_to_cand[h] = ci;
}

__global__ void __launch_bounds__(256) cand_keep_kernel(const int32_t* __restrict__ cand_nhits, int capacity, int min_hits,
                                                        const int32_t* __restrict__ cand_offsets, int n_events,
                                                        uint8_t* __restrict__ cand_keep) {
    const int total = min(cand_offsets[n_events], capacity);
    for (int ci = blockIdx.x * blockDim.x + threadIdx.x; ci < capacity; ci += gridDim.x * blockDim.x)
        cand_keep[ci] = (ci < total && cand_nhits[ci] >= min_hits) ? 1 : 0;
}

__global__ void __launch_bounds__(256) unassign_kernel(int n_hits, const uint8_t* __restrict__ cand_keep,
                                                       int32_t* __restrict__ hit_to_cand) {
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= n_hits) return;
    const int ci = hit_to_cand[h];
    if (ci >= 0 && !cand_keep[ci]) hit_to_cand[h] = -1;
}

// D12 decode: only hits left without a candidate take the key of the re-assignment round.  BY_BIN: the key's low word
// is ~(linear bin) (column walk); else ~(candidate index) (full scan).
template <bool BY_BIN>
__global__ void __launch_bounds__(256) reassign_decode_kernel(HoughConsts c, const unsigned long long* __restrict__ best_key,
                                                              int n_hits, const int32_t* __restrict__ off, int n_events,
                                                              const hough_candidate* __restrict__ cands,
                                                              const int32_t* __restrict__ cand_offsets, int capacity,
                                                              int32_t* __restrict__ hit_to_cand,
                                                              int32_t* __restrict__ cand_nhits) {
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= n_hits) return;
    if (hit_to_cand[h] >= 0) return;
    const unsigned long long key = best_key[h];
    if (!key) return;
    const unsigned low = 0xFFFFFFFFu - (unsigned)(key & 0xFFFFFFFFull);
    int ci = (int)low;
    if (BY_BIN) {
        const int e = find_event_a(off, n_events, h);
        int lo = min(__ldg(cand_offsets + e), capacity), hi = min(__ldg(cand_offsets + e + 1), capacity);
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            const int4 q = __ldg(reinterpret_cast<const int4*>(cands + mid));
            const unsigned lm = (unsigned)(q.y * c.n_phi + q.z) * (unsigned)c.n_qpt + (unsigned)q.w;
            if (lm < low) lo = mid + 1; else hi = mid;
        }
        ci = lo;
    }
    hit_to_cand[h] = ci;
    atomicAdd(cand_nhits + ci, 1);
}

}  // namespace

extern "C" int hough_assign_hits(hough_plan* p, const float* d_hits_xy, int32_t n_hits, const int32_t* d_event_offsets,
                                 int32_t n_events, const hough_candidate* d_cands, const int32_t* d_cand_offsets,
                                 int32_t capacity, int32_t assoc_dj, int32_t min_hits, int32_t* d_hit_to_cand,
                                 int32_t* d_cand_nhits, uint8_t* d_cand_keep, void* cuda_stream) {
    if (!p || !d_event_offsets || !d_cand_offsets) return HOUGH_ERR_INVALID_ARG;
    if (n_hits < 0 || n_events < 0 || n_hits > p->max_hits || n_events > p->max_events) return HOUGH_ERR_INVALID_ARG;
    if (capacity < 0 || assoc_dj < 0 || assoc_dj > 15) return HOUGH_ERR_INVALID_ARG;
    if (n_hits > 0 && (!d_hits_xy || !d_hit_to_cand)) return HOUGH_ERR_INVALID_ARG;
    if (capacity > 0 && (!d_cands || !d_cand_nhits || !d_cand_keep)) return HOUGH_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(d_hits_xy) & 7u) || (reinterpret_cast<uintptr_t>(d_cands) & 15u))
        return HOUGH_ERR_INVALID_ARG;
    if (n_events == 0) return n_hits == 0 ? HOUGH_OK : HOUGH_ERR_INVALID_ARG;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const bool tiled = !p->fullscan && p->tile_max_cols >= 1;
    if (capacity > 0) HOUGH_CUDA_TRY(cudaMemsetAsync(d_cand_nhits, 0, sizeof(int32_t) * (size_t)capacity, st));
    if (n_hits > 0) HOUGH_CUDA_TRY(cudaMemsetAsync(p->d_best_key, 0, sizeof(unsigned long long) * (size_t)n_hits, st));
    if (tiled) {
        bool by_index = false;
        if (n_hits > 0 && capacity > 0) {
            int rc = hough_stage_hits(p, d_hits_xy, n_hits, d_event_offsets, n_events, st, true);
            if (rc != HOUGH_OK) return rc;
            by_index = p->d_assoc_tab != nullptr && p->assign_candidates;
            if (by_index) {
                // plan option "assign_candidates": candidate-centric association (assoc.cu), keys carry the candidate index
                rc = hough_assoc_candidates(p, d_event_offsets, n_hits, n_events, d_cands, d_cand_offsets, capacity, assoc_dj,
                                            d_hit_to_cand, d_cand_nhits, st, nullptr);
                if (rc != HOUGH_OK) return rc;
            } else {
                WalkArgs a{};
                a.staged = p->d_staged;
                a.off = d_event_offsets;
                a.key_start = p->d_stage_cnt;
                walk_shape(p, n_events, a.n_slabs, a.slab_cols);
                a.stride = p->tile_stride_words;
                a.cands = d_cands;
                a.slice = p->d_slice;
                a.assoc_dj = assoc_dj;
                a.best_key = p->d_best_key;
                const long long tiles = (long long)n_events * p->c.n_d0 * a.n_slabs;
                if (tiles > (long long)p->slice_len) return HOUGH_ERR_UNSUPPORTED;
                cand_slice_kernel<<<(unsigned)((tiles + 255) / 256), 256, 0, st>>>(p->c, d_cands, d_cand_offsets, n_events,
                                                                                    capacity, a.n_slabs, a.slab_cols, p->d_slice);
                HOUGH_CUDA_TRY(cudaGetLastError());
                hough_count_launches(1);
                rc = walk_dispatch<WALK_ASSIGN>(p, n_events, a, p->tile32 != 0, false, st);
                if (rc != HOUGH_OK) return rc;
            }
        }
        if (n_hits > 0) {
            if (!by_index) {
                assign_decode_bin_kernel<<<(n_hits + 255) / 256, 256, 0, st>>>(p->c, p->d_best_key, n_hits, d_event_offsets,
                                                                               n_events, d_cands, d_cand_offsets, capacity,
                                                                               d_hit_to_cand, d_cand_nhits);
                HOUGH_CUDA_TRY(cudaGetLastError());
                hough_count_launches(1);
            }
        }
    } else {
        const size_t n_words = (size_t)n_events * p->c.words_per_event;
        HOUGH_CUDA_TRY(cudaMemsetAsync(p->d_mask, 0, sizeof(uint32_t) * n_words, st));
        if (capacity > 0) {
            const int blocks = min((capacity + 255) / 256, p->sm_count * 8);
            cand_index_kernel<<<blocks, 256, 0, st>>>(p->c, d_cands, d_cand_offsets, n_events, capacity, p->d_mask,
                                                      p->d_word_rank);
            HOUGH_CUDA_TRY(cudaGetLastError());
            hough_count_launches(1);
        }
        if (n_hits > 0) {
            const float2* hits = reinterpret_cast<const float2*>(d_hits_xy);
            const long long threads = (long long)n_hits * p->c.n_phi;
            const long long blocks = (threads + 255) / 256;
            if (blocks > 0x7fffffffLL) return HOUGH_ERR_UNSUPPORTED;
            if (capacity > 0) {
                assign_fullscan_kernel<<<(unsigned)blocks, 256, 0, st>>>(p->c, hits, n_hits, d_event_offsets, n_events, d_cands,
                                                                         p->d_mask, p->d_word_rank, assoc_dj, nullptr, p->d_best_key);
                HOUGH_CUDA_TRY(cudaGetLastError());
                hough_count_launches(1);
            }
            assign_decode_kernel<<<(n_hits + 255) / 256, 256, 0, st>>>(p->d_best_key, n_hits, d_hit_to_cand, d_cand_nhits);
            HOUGH_CUDA_TRY(cudaGetLastError());
            hough_count_launches(1);
        }
    }
    if (capacity > 0) {
        const int blocks = min((capacity + 255) / 256, p->sm_count * 8);
        cand_keep_kernel<<<blocks, 256, 0, st>>>(d_cand_nhits, capacity, min_hits, d_cand_offsets, n_events, d_cand_keep);
        HOUGH_CUDA_TRY(cudaGetLastError());
        hough_count_launches(1);
        if (n_hits > 0) {
            unassign_kernel<<<(n_hits + 255) / 256, 256, 0, st>>>(n_hits, d_cand_keep, d_hit_to_cand);
            HOUGH_CUDA_TRY(cudaGetLastError());
            hough_count_launches(1);
        }
    }
    return HOUGH_OK;
}


// D12: one re-assignment round after hough_assign_hits.  A kept candidate only gains hits, so the kept
// set does not change and this round is the fixed point of the rounds.
extern "C" int hough_reassign_hits(hough_plan* p, const float* d_hits_xy, int32_t n_hits, const int32_t* d_event_offsets,
                                   int32_t n_events, const hough_candidate* d_cands, const int32_t* d_cand_offsets,
                                   int32_t capacity, int32_t assoc_dj, int32_t max_rounds, int32_t* d_hit_to_cand,
                                   int32_t* d_cand_nhits, const uint8_t* d_cand_keep, void* cuda_stream) {
    if (!p || !d_event_offsets || !d_cand_offsets) return HOUGH_ERR_INVALID_ARG;
    if (n_hits < 0 || n_events < 0 || n_hits > p->max_hits || n_events > p->max_events) return HOUGH_ERR_INVALID_ARG;
    if (capacity < 0 || assoc_dj < 0 || assoc_dj > 15 || max_rounds < 1) return HOUGH_ERR_INVALID_ARG;
    if (n_hits > 0 && (!d_hits_xy || !d_hit_to_cand)) return HOUGH_ERR_INVALID_ARG;
    if (capacity > 0 && (!d_cands || !d_cand_nhits || !d_cand_keep)) return HOUGH_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(d_hits_xy) & 7u) || (reinterpret_cast<uintptr_t>(d_cands) & 15u))
        return HOUGH_ERR_INVALID_ARG;
    if (n_events == 0) return n_hits == 0 ? HOUGH_OK : HOUGH_ERR_INVALID_ARG;
    if (max_rounds < 2 || n_hits == 0 || capacity == 0) return HOUGH_OK;       // one round is D9 itself
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const bool tiled = !p->fullscan && p->tile_max_cols >= 1;
    HOUGH_CUDA_TRY(cudaMemsetAsync(p->d_best_key, 0, sizeof(unsigned long long) * (size_t)n_hits, st));
    if (tiled) {
        int rc = hough_stage_hits(p, d_hits_xy, n_hits, d_event_offsets, n_events, st, true);
        if (rc != HOUGH_OK) return rc;
        if (!p->reassign_walk && !p->d_assoc_tab && !p->assoc_tab_tried) {
            // No table yet and plan option "prepare_reassign" was not used.  Building it allocates and synchronises, which a
            // stream under capture forbids: build only when `st` is not capturing, otherwise this call re-walks the columns
            // (same results) and a later un-captured call builds.  A failed build is not an error either: walk instead.
            cudaStreamCaptureStatus cs = cudaStreamCaptureStatusActive;
            if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { (void)cudaGetLastError(); cs = cudaStreamCaptureStatusActive; }
            if (cs == cudaStreamCaptureStatusNone) hough_prepare_reassign(p);
        }
        if (p->d_assoc_tab != nullptr && !p->reassign_walk)
            // few candidates survive D9: the candidate-centric association (assoc.cu) visits only them
            return hough_assoc_candidates(p, d_event_offsets, n_hits, n_events, d_cands, d_cand_offsets, capacity, assoc_dj,
                                          d_hit_to_cand, d_cand_nhits, st, d_cand_keep);
        WalkArgs a{};
        a.staged = p->d_staged;
        a.off = d_event_offsets;
        a.key_start = p->d_stage_cnt;
        walk_shape(p, n_events, a.n_slabs, a.slab_cols);
        a.stride = p->tile_stride_words;
        a.cands = d_cands;
        a.slice = p->d_slice;
        a.assoc_dj = assoc_dj;
        a.best_key = p->d_best_key;
        a.keep = d_cand_keep;
        const long long tiles = (long long)n_events * p->c.n_d0 * a.n_slabs;
        if (tiles > (long long)p->slice_len) return HOUGH_ERR_UNSUPPORTED;
        cand_slice_kernel<<<(unsigned)((tiles + 255) / 256), 256, 0, st>>>(p->c, d_cands, d_cand_offsets, n_events, capacity,
                                                                            a.n_slabs, a.slab_cols, p->d_slice);
        HOUGH_CUDA_TRY(cudaGetLastError());
        rc = walk_dispatch<WALK_ASSIGN>(p, n_events, a, p->tile32 != 0, false, st);
        if (rc != HOUGH_OK) return rc;
        reassign_decode_kernel<true><<<(n_hits + 255) / 256, 256, 0, st>>>(p->c, p->d_best_key, n_hits, d_event_offsets, n_events,
                                                                           d_cands, d_cand_offsets, capacity, d_hit_to_cand,
                                                                           d_cand_nhits);
        HOUGH_CUDA_TRY(cudaGetLastError());
        hough_count_launches(2);
        return HOUGH_OK;
    }
    const size_t n_words = (size_t)n_events * p->c.words_per_event;
    HOUGH_CUDA_TRY(cudaMemsetAsync(p->d_mask, 0, sizeof(uint32_t) * n_words, st));
    const int blocks_c = min((capacity + 255) / 256, p->sm_count * 8);
    cand_index_kernel<<<blocks_c, 256, 0, st>>>(p->c, d_cands, d_cand_offsets, n_events, capacity, p->d_mask, p->d_word_rank);
    HOUGH_CUDA_TRY(cudaGetLastError());
    const float2* hits = reinterpret_cast<const float2*>(d_hits_xy);
    const long long blocks = ((long long)n_hits * p->c.n_phi + 255) / 256;
    if (blocks > 0x7fffffffLL) return HOUGH_ERR_UNSUPPORTED;
    assign_fullscan_kernel<<<(unsigned)blocks, 256, 0, st>>>(p->c, hits, n_hits, d_event_offsets, n_events, d_cands, p->d_mask,
                                                             p->d_word_rank, assoc_dj, d_cand_keep, p->d_best_key);
    HOUGH_CUDA_TRY(cudaGetLastError());
    reassign_decode_kernel<false><<<(n_hits + 255) / 256, 256, 0, st>>>(p->c, p->d_best_key, n_hits, d_event_offsets, n_events,
                                                                        d_cands, d_cand_offsets, capacity, d_hit_to_cand,
                                                                        d_cand_nhits);
    HOUGH_CUDA_TRY(cudaGetLastError());
    hough_count_launches(3);
    return HOUGH_OK;
}

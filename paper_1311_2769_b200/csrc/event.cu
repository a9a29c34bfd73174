// event.cu -- hough_event_run: the whole path of ONE small event of a two-parameter space in a single launch
// ("the two-parameter space presented here"; P:L55 / Fig. 2 is a time-per-event curve).
//
// A single event of a few hundred to a few thousand hits is launch-latency-bound on the general path (stage -> vote ->
// peaks -> assign is about 18 stream operations, 0.1 ms, for microseconds of work).  Here one thread-block CLUSTER does
// everything: CTA r of the cluster owns the phi0 columns [r * cols, (r + 1) * cols) of the accumulator as 16-bit bins in
// its shared memory, plus one halo column on each side (so the 3x3 peak test needs no neighbour CTA), and the steps are
// separated by cluster barriers instead of kernel boundaries:
//   0  zero the tile and this CTA's share of best_key / cand_nhits
//   1  vote: every CTA scans ALL hits of the event; a hit votes in the columns of its window that fall into the CTA's
//      slab (+ halo) with the prescribed D3 sequence (exact, no fast path: the event is small); shared-memory atomics
//   2  flush the slab to the global accumulator (the accumulator is an output of the path)
//   3  peaks: D5 test from the tile; count -> cluster barrier -> every CTA reads the other CTAs' counts through
//      distributed shared memory -> ordered emission of the records (D6, D7 centroid) and cand_offsets
//   4  association: the tile is reused as a presence map of the CTA's participating candidates; every CTA scans all hits
//      again and folds the D8 key of (hit, candidate) into best_key with atomicMax  -> cluster barrier
//   5  decode best_key -> hit_to_cand, count hits per candidate  -> cluster barrier
//   6  keep = nhits >= min_hits, hits of dropped candidates -> -1 (D9)
// Results are bit-identical to hough_vote + hough_find_peaks + hough_assign_hits (tests/test_gpu_event.py compares both
// with the CPU reference implementation under tests/).  Spaces with n_d0 > 1, tiles that do not fit 8 CTAs, or more than 2560 hits take those three
// calls instead (same results, more launches).
#include <algorithm>

#include <cooperative_groups.h>

#include "common.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int EV_THREADS = 1024;
constexpr int EV_MAX_CLUSTER = 8;                  // portable cluster size
constexpr size_t EV_SMEM_BUDGET = 200 * 1024;      // tile + hit cache bytes per CTA
constexpr long long EV_MAX_EVALS = 160000;         // hits x longest window above which the general path is faster
constexpr int EV_MAX_HITS = 2560;                 // hits of an event on the one-launch path (16-byte cache entry each)

struct EventArgs {
    const float2* hits;
    int n_hits;
    void* accum;
    int threshold;
    hough_candidate* cands;
    int capacity;
    int32_t* cand_off;                              // [2]
    int assoc_dj, min_hits;
    int32_t* h2c;
    int32_t* nhits;
    uint8_t* keep;
    unsigned long long* best_key;                   // [n_hits] plan workspace
    int cols_per_cta;
};

// column window of a hit in slice 0: first column and number of columns (stage.cu's classification, windows.cu's table)
__device__ __forceinline__ void ev_window(const HoughConsts& c, float x, float y, int& i_lo, int& steps) {
    const float r2 = d3_r2(x, y);
    int lo = 0, hi = c.n_class;                      // largest class with edge2[class] <= r2; NaN -> last class
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
    if (!(phi >= 0.0f && phi < c.two_pi_f)) phi = 0.0f;
    const float u = phi * c.u_scale - 0.5f;
    const int2 w = __ldg(c.win + (size_t)lo * c.n_d0);
    steps = min(w.y & 0x3fffffff, c.n_phi);
    i_lo = (int)ceilf(u + __int_as_float(w.x));
    if (i_lo < 0) i_lo += c.n_phi;
    if (i_lo >= c.n_phi) i_lo -= c.n_phi;
    if (!(i_lo >= 0 && i_lo < c.n_phi)) i_lo = 0;
}

__device__ __forceinline__ int ev_bin(const HoughConsts& c, float x, float y, float r2, int col) {
    const float2 cs = __ldg(c.cs + col);
    float w, f;
    d3_wf(x, y, cs.x, cs.y, w, f);
    if (!(f > 0.0f)) return -1;
    const float4 d = __ldg(c.d0t);
    return d3_bin_from_w(w, r2, d.x, d.y, d.z, c.A_f, c.qmin, c.inv_wq, c.nq_f, c.model != 0);
}

__device__ __forceinline__ void ev_tile_add(unsigned short* tile, int nq, int row, int j) {
    HOUGH_CHECK(row >= 0 && j >= 0 && j < nq);
    const unsigned idx = (unsigned)row * (unsigned)nq + (unsigned)j;
    atomicAdd(reinterpret_cast<unsigned*>(tile) + (idx >> 1), 1u << (16 * (idx & 1u)));
}

// D5 from the tile: rows r - 1, r, r + 1 are columns i - 1, i, i + 1 (halo rows close the circle), q/pT clipped
__device__ __forceinline__ bool ev_is_peak(const unsigned short* tile, int nq, int r, int j, int a) {
    bool peak = true;
#pragma unroll
    for (int di = -1; di <= 1; ++di) {
        const unsigned short* row = tile + (size_t)(r + di) * nq;
#pragma unroll
        for (int dj = -1; dj <= 1; ++dj) {
            const int jj = j + dj;
            if (jj < 0 || jj >= nq || (di == 0 && dj == 0)) continue;
            const int v = row[jj];
            const bool before = di < 0 || (di == 0 && dj < 0);
            peak = peak && (before ? (a > v) : (a >= v));
        }
    }
    return peak;
}

// exclusive prefix of `v` over the CTA's threads (in thread order) and the CTA total
__device__ __forceinline__ int ev_block_scan(int v, int* s_warp, int& total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    __syncthreads();                                 // s_warp free
    if (lane == 31) s_warp[warp] = x;
    __syncthreads();
    int pre = 0, tot = 0;
    for (int w = 0; w < EV_THREADS / 32; ++w) {
        const int s = s_warp[w];
        if (w < warp) pre += s;
        tot += s;
    }
    total = tot;
    return pre + x - v;
}

__global__ void __launch_bounds__(EV_THREADS, 1) event_kernel(const __grid_constant__ HoughConsts c, const __grid_constant__ EventArgs a) {
    extern __shared__ __align__(16) unsigned char ev_smem[];
    __shared__ int s_warp[EV_THREADS / 32];
    __shared__ int s_count;                          // peaks of this CTA (read by the other CTAs of the cluster)
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank(), C = (int)cluster.num_blocks();
    const int tid = threadIdx.x;
    const int nphi = c.n_phi, nq = c.n_qpt;
    const int c0 = rank * a.cols_per_cta;
    const int cols = max(min(a.cols_per_cta, nphi - c0), 0);
    float4* s_hit = reinterpret_cast<float4*>(ev_smem);                      // per hit {x, y, bits(first window column), bits(columns)}
    unsigned short* tile = reinterpret_cast<unsigned short*>(ev_smem + (size_t)a.n_hits * 16);   // rows 0 .. cols + 1: columns c0 - 1 .. c0 + cols
    const int tile_bins = (cols + 2) * nq;
    const int halo_l = c0 == 0 ? nphi - 1 : c0 - 1;
    const int halo_r = c0 + cols >= nphi ? c0 + cols - nphi : c0 + cols;
    const int gtid = rank * EV_THREADS + tid, gthreads = C * EV_THREADS;

    // ---- 0: zero ----
    for (int x = tid; x < (tile_bins + 1) / 2; x += EV_THREADS) reinterpret_cast<unsigned*>(tile)[x] = 0u;
    for (int h = gtid; h < a.n_hits; h += gthreads) a.best_key[h] = 0ull;
    for (int ci = gtid; ci < a.capacity; ci += gthreads) a.nhits[ci] = 0;
    if (tid == 0) s_count = 0;
    for (int h = tid; h < a.n_hits; h += EV_THREADS) {      // window of every hit, once (class search + atan2f)
        const float2 p = __ldg(a.hits + h);
        int i_lo, steps;
        ev_window(c, p.x, p.y, i_lo, steps);
        s_hit[h] = make_float4(p.x, p.y, __int_as_float(i_lo), __int_as_float(steps));
    }
    __syncthreads();

    // ---- 1: vote.  A warp takes a hit, its lanes the tile rows k = 0 .. cols + 1 (column c0 - 1 + k, cyclic): row k is
    // in the hit's window iff the column's position t inside the window is below `steps` ----
    const int lane = tid & 31, warp = tid >> 5;
    if (cols > 0) {
        for (int h = warp; h < a.n_hits; h += EV_THREADS / 32) {
            const float4 hv = s_hit[h];
            const float r2 = d3_r2(hv.x, hv.y);
            const int i_lo = __float_as_int(hv.z), steps = __float_as_int(hv.w);
            int t0 = halo_l - i_lo;                      // window position of row 0's column
            if (t0 < 0) t0 += nphi;
            for (int k = lane; k < cols + 2; k += 32) {
                int t = t0 + k;                          // k <= n_phi + 1: up to two turns
                if (t >= nphi) t -= nphi;
                if (t >= nphi) t -= nphi;
                if (t >= steps) continue;
                int col = halo_l + k;
                if (col >= nphi) col -= nphi;
                if (col >= nphi) col -= nphi;
                HOUGH_CHECK(col >= 0 && col < nphi && k <= cols + 1);
                const int j = ev_bin(c, hv.x, hv.y, r2, col);
                if (j >= 0) ev_tile_add(tile, nq, k, j);
            }
        }
    }
    __syncthreads();

    // ---- 2: flush the slab (rows 1 .. cols) ----
    {
        const int own_bins = cols * nq;
        const unsigned short* src = tile + nq;
        if (c.is_u16) {
            unsigned short* g = reinterpret_cast<unsigned short*>(a.accum) + (size_t)c0 * nq;
            for (int x = tid; x < own_bins; x += EV_THREADS) g[x] = src[x];
        } else {
            int* g = reinterpret_cast<int*>(a.accum) + (size_t)c0 * nq;
            for (int x = tid; x < own_bins; x += EV_THREADS) g[x] = (int)src[x];
        }
    }

    // ---- 3: peaks.  Every thread owns a run of consecutive linear bins of the slab, so one CTA scan of the per-thread
    // counts gives ranks that ascend with the linear bin (D6).  Pass A: count ----
    const int own_bins = cols * nq;
    const int per = (own_bins + EV_THREADS - 1) / EV_THREADS;
    const int x_begin = min(tid * per, own_bins), x_end = min(x_begin + per, own_bins);
    int mine = 0;
    {
        int r = x_begin / nq + 1, j = x_begin - (r - 1) * nq;
        for (int x = x_begin; x < x_end; ++x) {
            const int v = tile[(size_t)r * nq + j];
            if (v >= a.threshold && ev_is_peak(tile, nq, r, j, v)) ++mine;
            if (++j == nq) { j = 0; ++r; }
        }
    }
    int cta_total;
    const int my_pre = ev_block_scan(mine, s_warp, cta_total);
    if (tid == 0) s_count = cta_total;
    cluster.sync();                                  // every CTA's count is in its shared memory
    int base = 0, total_all = 0;
    for (int r = 0; r < C; ++r) {
        const int cnt = *cluster.map_shared_rank(&s_count, r);
        if (r < rank) base += cnt;
        total_all += cnt;
    }
    if (rank == 0 && tid == 0) { a.cand_off[0] = 0; a.cand_off[1] = total_all; }
    // Pass B: emission of the thread's own peaks at ranks base + my_pre, ...
    const int cta_rank = cta_total;                  // peaks of this CTA
    if (mine > 0 && base + my_pre < a.capacity) {
        int grank = base + my_pre;
        int r = x_begin / nq + 1, j = x_begin - (r - 1) * nq;
        for (int x = x_begin; x < x_end; ++x) {
            const int v = tile[(size_t)r * nq + j];
            if (v >= a.threshold && ev_is_peak(tile, nq, r, j, v)) {
                if (grank < a.capacity) {
                    long long S = 0, Sj = 0, Si = 0;
#pragma unroll
                    for (int di = -1; di <= 1; ++di)
#pragma unroll
                        for (int dj = -1; dj <= 1; ++dj) {
                            const int jj = j + dj;
                            if (jj < 0 || jj >= nq) continue;
                            const int val = tile[(size_t)(r + di) * nq + jj];
                            S += val; Sj += (long long)val * dj; Si += (long long)val * di;
                        }
                    hough_write_candidate(c, a.cands + grank, 0, 0, c0 + r - 1, j, v, S, Sj, Si, 0);
                }
                ++grank;
            }
            if (++j == nq) { j = 0; ++r; }
        }
    }
    __threadfence();
    __syncthreads();                                 // this CTA's records are written; the tile is free

    // ---- 4: association.  Presence map of the CTA's participating candidates, then all hits again ----
    const int first = min(base, a.capacity), end = min(base + cta_rank, a.capacity);
    for (int x = tid; x < (tile_bins + 1) / 2; x += EV_THREADS) reinterpret_cast<unsigned*>(tile)[x] = 0u;
    __syncthreads();
    for (int ci = first + tid; ci < end; ci += EV_THREADS) {
        const int4 q = *reinterpret_cast<const int4*>(a.cands + ci);          // event, k, i, j (written by this CTA)
        HOUGH_CHECK(q.z >= c0 && q.z < c0 + cols && q.w >= 0 && q.w < nq);
        tile[(size_t)(q.z - c0 + 1) * nq + q.w] = 1;
    }
    __syncthreads();
    if (cols > 0 && end > first) {
        for (int h = warp; h < a.n_hits; h += EV_THREADS / 32) {
            const float4 hv = s_hit[h];
            const float r2 = d3_r2(hv.x, hv.y);
            const int i_lo = __float_as_int(hv.z), steps = __float_as_int(hv.w);
            int t0 = c0 - i_lo;                          // window position of the slab's first column
            if (t0 < 0) t0 += nphi;
            unsigned long long best = 0ull;
            for (int k = lane; k < cols; k += 32) {
                int t = t0 + k;
                if (t >= nphi) t -= nphi;
                if (t >= steps) continue;
                const int col = c0 + k;
                const int jh = ev_bin(c, hv.x, hv.y, r2, col);
                if (jh < 0) continue;
                const unsigned short* row = tile + (size_t)(k + 1) * nq;
                for (int jj = max(jh - a.assoc_dj, 0); jj <= min(jh + a.assoc_dj, nq - 1); ++jj) {
                    if (!row[jj]) continue;
                    int lo = first, hi = end;              // the candidate at (col, jj): records sorted by (i, j)
                    while (lo < hi) {
                        const int mid = (lo + hi) >> 1;
                        const int4 q = *reinterpret_cast<const int4*>(a.cands + mid);
                        if (q.z < col || (q.z == col && q.w < jj)) lo = mid + 1; else hi = mid;
                    }
                    const unsigned votes = (unsigned)a.cands[lo].votes;
                    const unsigned long long key = ((unsigned long long)votes << 40) |
                                                   ((unsigned long long)(255 - abs(jj - jh)) << 32) |
                                                   (unsigned long long)(0xFFFFFFFFu - (unsigned)lo);
                    best = key > best ? key : best;
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const unsigned long long other = __shfl_xor_sync(0xffffffffu, best, o);
                best = other > best ? other : best;
            }
            if (lane == 0 && best) atomicMax(a.best_key + h, best);
        }
    }
    __threadfence();
    cluster.sync();

    // ---- 5: decode ----
    for (int h = gtid; h < a.n_hits; h += gthreads) {
        const unsigned long long key = a.best_key[h];
        int ci = -1;
        if (key) {
            ci = (int)(0xFFFFFFFFu - (unsigned)(key & 0xFFFFFFFFull));
            atomicAdd(a.nhits + ci, 1);
        }
        a.h2c[h] = ci;
    }
    __threadfence();
    cluster.sync();

    // ---- 6: keep / unassign (D9) ----
    const int n_part = min(total_all, a.capacity);
    for (int ci = gtid; ci < a.capacity; ci += gthreads)
        a.keep[ci] = (ci < n_part && __ldcg(a.nhits + ci) >= a.min_hits) ? 1 : 0;
    for (int h = gtid; h < a.n_hits; h += gthreads) {
        const int ci = a.h2c[h];
        if (ci >= 0 && __ldcg(a.nhits + ci) < a.min_hits) a.h2c[h] = -1;
    }
}

}  // namespace

extern "C" int hough_event_run(hough_plan* p, const float* d_hits_xy, int32_t n_hits, const int32_t* d_event_offsets,
                               void* d_accum, int32_t threshold, hough_candidate* d_cands, int32_t capacity,
                               int32_t* d_cand_offsets, int32_t assoc_dj, int32_t min_hits, int32_t* d_hit_to_cand,
                               int32_t* d_cand_nhits, uint8_t* d_cand_keep, void* cuda_stream) {
    if (!p || !d_event_offsets || !d_accum || !d_cand_offsets) return HOUGH_ERR_INVALID_ARG;
    if (n_hits < 0 || n_hits > p->max_hits || capacity < 0 || assoc_dj < 0 || assoc_dj > 15) return HOUGH_ERR_INVALID_ARG;
    if (n_hits > 0 && (!d_hits_xy || !d_hit_to_cand)) return HOUGH_ERR_INVALID_ARG;
    if (capacity > 0 && (!d_cands || !d_cand_nhits || !d_cand_keep)) return HOUGH_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(d_hits_xy) & 7u) || (reinterpret_cast<uintptr_t>(d_cands) & 15u) ||
        (reinterpret_cast<uintptr_t>(d_accum) & 3u))
        return HOUGH_ERR_INVALID_ARG;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const HoughConsts& c = p->c;
    // cluster shape: the fewest CTAs whose tiles fit, then more (up to 8) while every CTA keeps at least 32 columns
    int n_cta = 0;
    const size_t hit_bytes = (size_t)std::max(n_hits, 0) * 16;
    // the cluster runs on at most 8 SMs: it wins while the event is latency-bound, i.e. while hits x columns per hit stays
    // small (measured break-even about 2e5 evaluations per phase; an upper estimate from the longest class window)
    const bool small = n_hits <= EV_MAX_HITS &&
                       (p->event_cluster || (long long)n_hits * std::max(p->event_max_steps, 1) <= EV_MAX_EVALS);
    if (c.n_d0 == 1 && small && !p->fullscan && !p->event_general) {
        for (int k = 1; k <= EV_MAX_CLUSTER; ++k) {
            const int cols = (c.n_phi + k - 1) / k;
            if ((size_t)(cols + 2) * c.n_qpt * 2 + 16 + hit_bytes <= EV_SMEM_BUDGET) { n_cta = k; break; }
        }
        // more CTAs than the tiles need: every per-bin pass (zero, flush, peaks) and the hit scans shrink with the slab
        while (n_cta > 0 && n_cta < EV_MAX_CLUSTER && (c.n_phi + n_cta) / (n_cta + 1) >= 16) ++n_cta;
    }
    // general path: the three calls (same results)
    auto general = [&]() -> int {
        int rc = hough_vote(p, d_hits_xy, n_hits, d_event_offsets, 1, d_accum, cuda_stream);
        if (rc != HOUGH_OK) return rc;
        rc = hough_find_peaks(p, d_accum, 1, threshold, d_cands, capacity, d_cand_offsets, cuda_stream);
        if (rc != HOUGH_OK) return rc;
        return hough_assign_hits(p, d_hits_xy, n_hits, d_event_offsets, 1, d_cands, d_cand_offsets, capacity, assoc_dj, min_hits,
                                 d_hit_to_cand, d_cand_nhits, d_cand_keep, cuda_stream);
    };
    if (n_cta == 0) return general();
    EventArgs a{};
    a.hits = reinterpret_cast<const float2*>(d_hits_xy);
    a.n_hits = n_hits;
    a.accum = d_accum;
    a.threshold = threshold;
    a.cands = d_cands;
    a.capacity = capacity;
    a.cand_off = d_cand_offsets;
    a.assoc_dj = assoc_dj;
    a.min_hits = min_hits;
    a.h2c = d_hit_to_cand;
    a.nhits = d_cand_nhits;
    a.keep = d_cand_keep;
    a.best_key = p->d_best_key;
    a.cols_per_cta = (c.n_phi + n_cta - 1) / n_cta;
    const size_t smem = (hit_bytes + (size_t)(a.cols_per_cta + 2) * c.n_qpt * 2 + 15) & ~(size_t)15;
    static size_t smem_configured[HOUGH_MAX_DEVICES] = {};
    const int dev = p->device >= 0 && p->device < HOUGH_MAX_DEVICES ? p->device : 0;
    if (smem > smem_configured[dev] || p->device >= HOUGH_MAX_DEVICES) {
        HOUGH_CUDA_TRY(cudaFuncSetAttribute(event_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)EV_SMEM_BUDGET));
        smem_configured[dev] = EV_SMEM_BUDGET;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)n_cta, 1, 1);
    cfg.blockDim = dim3(EV_THREADS, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)n_cta;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    // Can a cluster of n_cta such CTAs be co-scheduled on this device at all?  (Not under every MIG / MPS partition, nor on a
    // GPC with fewer free SMs.)  Asked once per (device, cluster size) with the largest shared-memory block the path uses;
    // 0 clusters, a failing query or a failing launch send this and later such calls to the general path: same results.
    static signed char cluster_ok[HOUGH_MAX_DEVICES][EV_MAX_CLUSTER + 1] = {};       // 0: not asked, 1: fits, -1: does not
    signed char& ok = cluster_ok[dev][n_cta];
    if (ok == 0 || p->device >= HOUGH_MAX_DEVICES) {
        cudaLaunchConfig_t q = cfg;
        q.dynamicSmemBytes = EV_SMEM_BUDGET;
        int n_clusters = 0;
        if (cudaOccupancyMaxActiveClusters(&n_clusters, event_kernel, &q) != cudaSuccess) { (void)cudaGetLastError(); n_clusters = 0; }
        ok = n_clusters > 0 ? 1 : -1;
    }
    if (ok < 0) return general();
    if (cudaLaunchKernelEx(&cfg, event_kernel, c, a) != cudaSuccess) {
        (void)cudaGetLastError();
        ok = -1;
        return general();
    }
    hough_count_launches(1);
    return HOUGH_OK;
}

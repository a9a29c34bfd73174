// pipeline.cu -- A6: batched multi-event path (B:L5 "a batched multi-event path using CUDA streams and graphs";
// B:L10 "one accumulator per event, reused across event tiles on 4 CUDA streams").
//
// hough_pipeline_run_host cuts the events into tiles of `tile_events`, deals the tiles round-robin to `n_streams`
// lanes (stream + plan + accumulator + device buffers of ONE tile) and, per tile, runs
//     H2D hits, offsets -> hough_vote -> hough_find_peaks -> hough_assign_hits -> D2H per-event counts      (part A)
//     [host: the tile's candidate base is the sum of the totals of all earlier tiles]
//     rebase kernel (tile-local -> global event and candidate indices) -> D2H hit_to_cand, records, nhits, keep   (part B)
// Part A of a lane is captured as a CUDA graph the first time and re-captured + cudaGraphExecUpdate'd for the
// following tiles of that lane (same topology, other sizes), then launched with one cudaGraphLaunch.  Part B of tile
// t is issued when tile t + n_streams is about to reuse the lane, so n_streams - 1 tiles are always in flight while
// the host waits for a count.  Host buffers should be pinned (copies are cudaMemcpyAsync).
#include <algorithm>
#include <cstring>
#include <new>
#include <vector>

#include "common.cuh"

namespace {

__global__ void __launch_bounds__(256) rebase_kernel(int32_t* __restrict__ hit_to_cand, int n_hits, int cand_base,
                                                     hough_candidate* __restrict__ cands, int n_cands, int event_base) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n_hits) {
        const int c = hit_to_cand[t];
        if (c >= 0) hit_to_cand[t] = c + cand_base;
    }
    if (t < n_cands) cands[t].event += event_base;
}

// ---- "kept_only" mode: compact the candidates that survive duplicate removal (D9) on the device -------------------
constexpr int KEEP_BLOCK = 4096;                      // candidates per compaction block (256 threads x 16)

// kept candidates per block of KEEP_BLOCK; n_c = min(cand_off[n_ev], cap) is read on the device
__global__ void __launch_bounds__(256) keep_count_kernel(const uint8_t* __restrict__ keep, const int32_t* __restrict__ cand_off,
                                                         int n_ev, int cap, int32_t* __restrict__ blk) {
    const int n_c = min(cand_off[n_ev], cap);
    const int base = blockIdx.x * KEEP_BLOCK + threadIdx.x * 16;
    int cnt = 0;
    if (base + 16 <= n_c) {
        const uint4 q = *reinterpret_cast<const uint4*>(keep + base);            // flags are 0 / 1
        cnt = __popc(q.x) + __popc(q.y) + __popc(q.z) + __popc(q.w);
    } else {
        for (int c = base; c < min(base + 16, n_c); ++c) cnt += keep[c];
    }
    cnt = __reduce_add_sync(0xffffffffu, cnt);
    __shared__ int s[8];
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = cnt;
    __syncthreads();
    if (threadIdx.x == 0) blk[blockIdx.x] = s[0] + s[1] + s[2] + s[3] + s[4] + s[5] + s[6] + s[7];
}

__global__ void __launch_bounds__(1024) keep_scan_kernel(int32_t* blk, int n_blk) {
    cta_exclusive_scan(blk, n_blk, blk + n_blk);          // blk[n_blk] = kept candidates of the tile
}

// pre[c] = kept candidates before c (for every c < n_c); kept records and their hit counts move to rank pre[c]
__global__ void __launch_bounds__(256) keep_compact_kernel(const uint8_t* __restrict__ keep, const int32_t* __restrict__ cand_off,
                                                           int n_ev, int cap, const int32_t* __restrict__ blk,
                                                           const hough_candidate* __restrict__ cands, const int32_t* __restrict__ nh,
                                                           int32_t* __restrict__ pre, hough_candidate* __restrict__ kcands,
                                                           int32_t* __restrict__ knh) {
    const int n_c = min(cand_off[n_ev], cap);
    const int base = blockIdx.x * KEEP_BLOCK + threadIdx.x * 16;
    int cnt = 0;
    for (int c = base; c < min(base + 16, n_c); ++c) cnt += keep[c];
    int x = cnt;                                          // inclusive scan over the block's 256 threads
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, x, o);
        if ((threadIdx.x & 31) >= o) x += y;
    }
    __shared__ int s[8];
    if ((threadIdx.x & 31) == 31) s[threadIdx.x >> 5] = x;
    __syncthreads();
    int run = blk[blockIdx.x] + x - cnt;
    for (int w = 0; w < (int)(threadIdx.x >> 5); ++w) run += s[w];
    for (int c = base; c < min(base + 16, n_c); ++c) {
        pre[c] = run;
        if (keep[c]) {
            const int4* src = reinterpret_cast<const int4*>(cands + c);
            int4* dst = reinterpret_cast<int4*>(kcands + run);
            dst[0] = src[0];
            dst[1] = src[1];
            knh[run] = nh[c];
            ++run;
        }
    }
}

// per-event offsets of the kept list and hit -> kept rank (hits of dropped candidates are already -1, D9)
__global__ void __launch_bounds__(256) keep_finish_kernel(const int32_t* __restrict__ cand_off, int n_ev, int cap,
                                                          const int32_t* __restrict__ blk, int n_blk, const int32_t* __restrict__ pre,
                                                          int32_t* __restrict__ kept_off, int32_t* __restrict__ h2c, int n_hits) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int n_c = min(cand_off[n_ev], cap);
    if (t <= n_ev) {
        const int c = cand_off[t];
        kept_off[t] = c < n_c ? pre[c] : blk[n_blk];
    }
    if (t < n_hits) {
        const int c = h2c[t];
        if (c >= 0) h2c[t] = pre[c];
    }
}

struct Lane {
    cudaStream_t st = nullptr;
    hough_plan* plan = nullptr;
    void* d_accum = nullptr;
    float* d_hits = nullptr;
    int32_t* d_off = nullptr;
    hough_candidate* d_cands = nullptr;
    int32_t* d_cand_off = nullptr;
    int32_t* d_h2c = nullptr;
    int32_t* d_nh = nullptr;
    uint8_t* d_keep = nullptr;
    int32_t* h_off = nullptr;        // pinned: tile-relative event offsets
    int32_t* h_cand_off = nullptr;   // pinned: the tile's exclusive per-event candidate offsets
    // kept_only mode
    int32_t* d_pre = nullptr;        // [cap] kept candidates before each candidate
    int32_t* d_blk = nullptr;        // [cap / KEEP_BLOCK + 2]
    hough_candidate* d_kcands = nullptr;
    int32_t* d_knh = nullptr;
    int32_t* d_kept_off = nullptr;   // [tile_events + 1]
    int32_t* h_kept_off = nullptr;   // pinned
    cudaEvent_t counted = nullptr;
    cudaGraphExec_t exec = nullptr;
    bool warmed = false;             // first tile of a lane runs un-captured (lazy kernel attributes)
    // tile in flight
    int tile = -1, e0 = 0, e1 = 0, h0 = 0, h1 = 0;
};

}  // namespace

struct hough_pipeline {
    hough_binning b;
    int32_t tile_events, max_hits, tile_cap, n_streams;
    std::vector<Lane> lanes;
    int use_graphs;
    int kept_only;
    int reassign;                       // 1: hough_reassign_hits (D12) after the association of every tile
};

static void pipeline_free(hough_pipeline* p) {
    if (!p) return;
    for (Lane& l : p->lanes) {
        if (l.exec) cudaGraphExecDestroy(l.exec);
        if (l.counted) cudaEventDestroy(l.counted);
        if (l.plan) hough_plan_destroy(l.plan);
        cudaFree(l.d_accum); cudaFree(l.d_hits); cudaFree(l.d_off); cudaFree(l.d_cands); cudaFree(l.d_cand_off);
        cudaFree(l.d_h2c); cudaFree(l.d_nh); cudaFree(l.d_keep);
        if (l.h_off) cudaFreeHost(l.h_off);
        if (l.h_cand_off) cudaFreeHost(l.h_cand_off);
        cudaFree(l.d_pre); cudaFree(l.d_blk); cudaFree(l.d_kcands); cudaFree(l.d_knh); cudaFree(l.d_kept_off);
        if (l.h_kept_off) cudaFreeHost(l.h_kept_off);
        if (l.st) cudaStreamDestroy(l.st);
    }
    delete p;
}

extern "C" int hough_pipeline_create(const hough_binning* b, const hough_geometry* g, int32_t tile_events,
                                     int32_t max_hits_per_tile, int32_t tile_cand_capacity, int32_t n_streams,
                                     hough_pipeline** out) {
    if (!b || !g || !out) return HOUGH_ERR_INVALID_ARG;
    if (tile_events <= 0 || max_hits_per_tile <= 0 || tile_cand_capacity < 0 || n_streams <= 0 || n_streams > 64)
        return HOUGH_ERR_INVALID_ARG;
    hough_pipeline* p = new (std::nothrow) hough_pipeline();
    if (!p) return HOUGH_ERR_ALLOC;
    p->b = *b;
    p->tile_events = tile_events;
    p->max_hits = max_hits_per_tile;
    p->tile_cap = tile_cand_capacity;
    p->n_streams = n_streams;
    const char* env = getenv("HOUGH_PIPELINE_NO_GRAPHS");
    p->use_graphs = (env && env[0] == '1') ? 0 : 1;
    p->kept_only = 0;
    p->reassign = 0;
    p->lanes.resize(n_streams);
    int rc = HOUGH_OK;
    for (Lane& l : p->lanes) {
        rc = hough_plan_create(b, g, max_hits_per_tile, tile_events, &l.plan);
        if (rc != HOUGH_OK) break;
        hough_plan_set_option(l.plan, "reuse_staging", 1);   // vote and assign of a tile see the same device hits
        bool ok = cudaStreamCreateWithFlags(&l.st, cudaStreamNonBlocking) == cudaSuccess;
        ok = ok && cudaEventCreateWithFlags(&l.counted, cudaEventDisableTiming) == cudaSuccess;
        const size_t cap = (size_t)std::max(tile_cand_capacity, 1);
        ok = ok && cudaMalloc(&l.d_accum, hough_accum_bytes(l.plan, tile_events)) == cudaSuccess;
        ok = ok && cudaMalloc((void**)&l.d_hits, sizeof(float) * 2 * (size_t)max_hits_per_tile) == cudaSuccess;
        ok = ok && cudaMalloc((void**)&l.d_off, sizeof(int32_t) * ((size_t)tile_events + 1)) == cudaSuccess;
        ok = ok && cudaMalloc((void**)&l.d_cands, sizeof(hough_candidate) * cap) == cudaSuccess;
        ok = ok && cudaMalloc((void**)&l.d_cand_off, sizeof(int32_t) * ((size_t)tile_events + 1)) == cudaSuccess;
        ok = ok && cudaMalloc((void**)&l.d_h2c, sizeof(int32_t) * (size_t)max_hits_per_tile) == cudaSuccess;
        ok = ok && cudaMalloc((void**)&l.d_nh, sizeof(int32_t) * cap) == cudaSuccess;
        ok = ok && cudaMalloc((void**)&l.d_keep, cap) == cudaSuccess;
        ok = ok && cudaMallocHost((void**)&l.h_off, sizeof(int32_t) * ((size_t)tile_events + 1)) == cudaSuccess;
        ok = ok && cudaMallocHost((void**)&l.h_cand_off, sizeof(int32_t) * ((size_t)tile_events + 1)) == cudaSuccess;
        if (!ok) { (void)cudaGetLastError(); rc = HOUGH_ERR_ALLOC; break; }
    }
    if (rc != HOUGH_OK) { pipeline_free(p); return rc; }
    *out = p;
    return HOUGH_OK;
}

extern "C" int hough_pipeline_set_option(hough_pipeline* p, const char* key, int32_t value) {
    if (!p || !key) return HOUGH_ERR_INVALID_ARG;
    if (strcmp(key, "graphs") == 0) { p->use_graphs = value ? 1 : 0; return HOUGH_OK; }
    if (strcmp(key, "reassign") == 0) {
        p->reassign = value ? 1 : 0;
        if (value && !p->lanes.empty()) {
            // The D12 round's azimuth table is built HERE, never inside a tile's (captured) sequence: once, on lane 0's plan;
            // the other lanes' plans have the same binning and geometry and borrow it (read-only).  No table (it does not
            // fit, or the build failed): every lane re-walks the vote columns instead.
            hough_plan* first = p->lanes[0].plan;
            hough_prepare_reassign(first);
            for (size_t i = 1; i < p->lanes.size(); ++i) {
                hough_plan* q = p->lanes[i].plan;
                if (q->d_assoc_tab || q->assoc_tab_tried) continue;
                q->assoc_tab_tried = 1;
                q->d_assoc_tab = first->d_assoc_tab;
                q->assoc_tab_borrowed = first->d_assoc_tab != nullptr;
            }
        }
        for (Lane& l : p->lanes) {                           // another node list: the lanes' graphs are rebuilt, and the next
            if (l.exec) { cudaGraphExecDestroy(l.exec); l.exec = nullptr; }      // tile of a lane runs un-captured once (lazy
            l.warmed = false;                                                    // kernel attributes of the added kernels)
        }
        return HOUGH_OK;
    }
    if (strcmp(key, "kept_only") != 0) return HOUGH_ERR_INVALID_ARG;
    if (value && !p->lanes.empty() && !p->lanes[0].d_pre) {          // buffers of the compaction, once
        const size_t cap = (size_t)std::max(p->tile_cap, 1);
        for (Lane& l : p->lanes) {
            bool ok = cudaMalloc((void**)&l.d_pre, sizeof(int32_t) * cap) == cudaSuccess;
            ok = ok && cudaMalloc((void**)&l.d_blk, sizeof(int32_t) * (cap / KEEP_BLOCK + 2)) == cudaSuccess;
            ok = ok && cudaMalloc((void**)&l.d_kcands, sizeof(hough_candidate) * cap) == cudaSuccess;
            ok = ok && cudaMalloc((void**)&l.d_knh, sizeof(int32_t) * cap) == cudaSuccess;
            ok = ok && cudaMalloc((void**)&l.d_kept_off, sizeof(int32_t) * ((size_t)p->tile_events + 1)) == cudaSuccess;
            ok = ok && cudaMallocHost((void**)&l.h_kept_off, sizeof(int32_t) * ((size_t)p->tile_events + 1)) == cudaSuccess;
            if (!ok) { (void)cudaGetLastError(); return HOUGH_ERR_ALLOC; }
        }
    }
    p->kept_only = value ? 1 : 0;
    for (Lane& l : p->lanes) {                           // another node list: the lanes' graphs are rebuilt
        if (l.exec) { cudaGraphExecDestroy(l.exec); l.exec = nullptr; }
    }
    return HOUGH_OK;
}

extern "C" int hough_pipeline_destroy(hough_pipeline* p) {
    if (!p) return HOUGH_ERR_INVALID_ARG;
    pipeline_free(p);
    return HOUGH_OK;
}

// part A of one tile on its lane's stream: copies in, the three calls, counts out
static int enqueue_part_a(hough_pipeline* p, Lane& l, const float* h_hits_xy, int32_t threshold, int32_t assoc_dj,
                          int32_t min_hits) {
    const int n_ev = l.e1 - l.e0, n_h = l.h1 - l.h0;
    if (n_h > 0)
        HOUGH_CUDA_TRY(cudaMemcpyAsync(l.d_hits, h_hits_xy + 2 * (size_t)l.h0, sizeof(float) * 2 * (size_t)n_h,
                                       cudaMemcpyHostToDevice, l.st));
    HOUGH_CUDA_TRY(cudaMemcpyAsync(l.d_off, l.h_off, sizeof(int32_t) * ((size_t)n_ev + 1), cudaMemcpyHostToDevice, l.st));
    int rc = hough_vote(l.plan, l.d_hits, n_h, l.d_off, n_ev, l.d_accum, l.st);
    if (rc != HOUGH_OK) return rc;
    rc = hough_find_peaks(l.plan, l.d_accum, n_ev, threshold, p->tile_cap > 0 ? l.d_cands : nullptr, p->tile_cap, l.d_cand_off,
                          l.st);
    if (rc != HOUGH_OK) return rc;
    rc = hough_assign_hits(l.plan, l.d_hits, n_h, l.d_off, n_ev, l.d_cands, l.d_cand_off, p->tile_cap, assoc_dj, min_hits,
                           l.d_h2c, l.d_nh, l.d_keep, l.st);
    if (rc != HOUGH_OK) return rc;
    if (p->reassign && p->tile_cap > 0) {                // D12: orphan hits take the best surviving candidate
        rc = hough_reassign_hits(l.plan, l.d_hits, n_h, l.d_off, n_ev, l.d_cands, l.d_cand_off, p->tile_cap, assoc_dj, 2, l.d_h2c,
                                 l.d_nh, l.d_keep, l.st);
        if (rc != HOUGH_OK) return rc;
    }
    HOUGH_CUDA_TRY(cudaMemcpyAsync(l.h_cand_off, l.d_cand_off, sizeof(int32_t) * ((size_t)n_ev + 1), cudaMemcpyDeviceToHost,
                                   l.st));
    if (p->kept_only && p->tile_cap > 0) {
        const int n_blk = p->tile_cap / KEEP_BLOCK + 1;
        keep_count_kernel<<<n_blk, 256, 0, l.st>>>(l.d_keep, l.d_cand_off, n_ev, p->tile_cap, l.d_blk);
        keep_scan_kernel<<<1, 1024, 0, l.st>>>(l.d_blk, n_blk);
        keep_compact_kernel<<<n_blk, 256, 0, l.st>>>(l.d_keep, l.d_cand_off, n_ev, p->tile_cap, l.d_blk, l.d_cands, l.d_nh, l.d_pre,
                                                     l.d_kcands, l.d_knh);
        const int n_thr = std::max(n_h, n_ev + 1);
        keep_finish_kernel<<<(n_thr + 255) / 256, 256, 0, l.st>>>(l.d_cand_off, n_ev, p->tile_cap, l.d_blk, n_blk, l.d_pre,
                                                                 l.d_kept_off, l.d_h2c, n_h);
        HOUGH_CUDA_TRY(cudaGetLastError());
        hough_count_launches(4);
        HOUGH_CUDA_TRY(cudaMemcpyAsync(l.h_kept_off, l.d_kept_off, sizeof(int32_t) * ((size_t)n_ev + 1), cudaMemcpyDeviceToHost,
                                       l.st));
    }
    return HOUGH_OK;
}

static int launch_part_a(hough_pipeline* p, Lane& l, const float* h_hits_xy, int32_t threshold, int32_t assoc_dj,
                         int32_t min_hits) {
    if (!p->use_graphs || !l.warmed) {
        l.warmed = true;
        return enqueue_part_a(p, l, h_hits_xy, threshold, assoc_dj, min_hits);
    }
    // capture the tile's sequence, then update the lane's executable graph in place (same topology, other sizes)
    HOUGH_CUDA_TRY(cudaStreamBeginCapture(l.st, cudaStreamCaptureModeThreadLocal));
    const int rc = enqueue_part_a(p, l, h_hits_xy, threshold, assoc_dj, min_hits);
    cudaGraph_t graph = nullptr;
    const cudaError_t ce = cudaStreamEndCapture(l.st, &graph);
    if (rc != HOUGH_OK || ce != cudaSuccess || !graph) {
        if (graph) cudaGraphDestroy(graph);
        (void)cudaGetLastError();
        if (rc != HOUGH_OK) return rc;
        p->use_graphs = 0;                               // capture not possible here: plain launches from now on
        return enqueue_part_a(p, l, h_hits_xy, threshold, assoc_dj, min_hits);
    }
    bool ready = false;
    if (l.exec) {
        cudaGraphExecUpdateResultInfo info;
        if (cudaGraphExecUpdate(l.exec, graph, &info) == cudaSuccess) ready = true;
        else { (void)cudaGetLastError(); cudaGraphExecDestroy(l.exec); l.exec = nullptr; }
    }
    if (!ready) {
        if (cudaGraphInstantiate(&l.exec, graph, 0) != cudaSuccess) {
            hough_set_last_cuda_error(cudaGetLastError(), "cudaGraphInstantiate");
            cudaGraphDestroy(graph);
            return HOUGH_ERR_CUDA;
        }
    }
    cudaGraphDestroy(graph);
    HOUGH_CUDA_TRY(cudaGraphLaunch(l.exec, l.st));
    return HOUGH_OK;
}

extern "C" int hough_pipeline_run_host(hough_pipeline* p, const float* h_hits_xy, int32_t n_hits,
                                       const int32_t* h_event_offsets, int32_t n_events, int32_t threshold,
                                       int32_t assoc_dj, int32_t min_hits, int32_t* h_hit_to_cand,
                                       int32_t* h_cand_offsets, hough_candidate* h_cands, int32_t cand_capacity,
                                       int32_t* h_cand_nhits, uint8_t* h_cand_keep, int32_t* h_overflowed) {
    if (!p || !h_event_offsets || !h_cand_offsets) return HOUGH_ERR_INVALID_ARG;
    if (n_hits < 0 || n_events < 0 || cand_capacity < 0 || assoc_dj < 0 || assoc_dj > 15) return HOUGH_ERR_INVALID_ARG;
    if (n_hits > 0 && (!h_hits_xy || !h_hit_to_cand)) return HOUGH_ERR_INVALID_ARG;
    if (cand_capacity > 0 && (!h_cands || !h_cand_nhits || !h_cand_keep)) return HOUGH_ERR_INVALID_ARG;
    if (h_event_offsets[0] != 0 || h_event_offsets[n_events] != n_hits) return HOUGH_ERR_INVALID_ARG;
    if (h_overflowed) *h_overflowed = 0;
    h_cand_offsets[0] = 0;
    const int n_tiles = (n_events + p->tile_events - 1) / p->tile_events;
    const int S = p->n_streams;
    long long cand_base = 0;                             // global rank of the first candidate of the tile being finished
    int status = HOUGH_OK;

    // part B of the tile that lane `l` carries: wait for its counts, rebase on the device, copy the results out
    auto finish = [&](Lane& l) -> int {
        if (l.tile < 0) return HOUGH_OK;
        HOUGH_CUDA_TRY(cudaEventSynchronize(l.counted));
        const int n_ev = l.e1 - l.e0, n_h = l.h1 - l.h0;
        const bool kept = p->kept_only && p->tile_cap > 0;
        const int32_t* toff = kept ? l.h_kept_off : l.h_cand_off;        // offsets of the list that goes to the caller
        if (l.h_cand_off[n_ev] > p->tile_cap && h_overflowed) *h_overflowed = 1;
        const int total = toff[n_ev];
        const int n_c = kept ? total : std::min(total, p->tile_cap);
        const hough_candidate* d_rec = kept ? l.d_kcands : l.d_cands;
        const int32_t* d_rnh = kept ? l.d_knh : l.d_nh;
        for (int i = 1; i <= n_ev; ++i)
            h_cand_offsets[l.e0 + i] = (int32_t)std::min<long long>(cand_base + toff[i], 0x7fffffffLL);
        // records that fit the caller's capacity
        const long long room = std::max<long long>(0, (long long)cand_capacity - cand_base);
        const int n_out = (int)std::min<long long>(n_c, room);
        if (n_c > n_out && h_overflowed) *h_overflowed = 1;
        const int n_thr = std::max(n_h, n_c);
        if (n_thr > 0) {
            rebase_kernel<<<(n_thr + 255) / 256, 256, 0, l.st>>>(l.d_h2c, n_h, (int)std::min<long long>(cand_base, 0x7fffffffLL),
                                                                const_cast<hough_candidate*>(d_rec), n_c, l.e0);
            HOUGH_CUDA_TRY(cudaGetLastError());
            hough_count_launches(1);
        }
        if (n_h > 0)
            HOUGH_CUDA_TRY(cudaMemcpyAsync(h_hit_to_cand + l.h0, l.d_h2c, sizeof(int32_t) * (size_t)n_h, cudaMemcpyDeviceToHost, l.st));
        if (n_out > 0) {
            HOUGH_CUDA_TRY(cudaMemcpyAsync(h_cands + cand_base, d_rec, sizeof(hough_candidate) * (size_t)n_out,
                                           cudaMemcpyDeviceToHost, l.st));
            HOUGH_CUDA_TRY(cudaMemcpyAsync(h_cand_nhits + cand_base, d_rnh, sizeof(int32_t) * (size_t)n_out, cudaMemcpyDeviceToHost, l.st));
            if (kept) memset(h_cand_keep + cand_base, 1, (size_t)n_out);        // every returned candidate is a kept one
            else HOUGH_CUDA_TRY(cudaMemcpyAsync(h_cand_keep + cand_base, l.d_keep, (size_t)n_out, cudaMemcpyDeviceToHost, l.st));
        }
        cand_base += total;
        l.tile = -1;
        return HOUGH_OK;
    };

    for (int t = 0; t < n_tiles && status == HOUGH_OK; ++t) {
        Lane& l = p->lanes[t % S];
        status = finish(l);                              // the lane's previous tile (t - S)
        if (status != HOUGH_OK) break;
        l.tile = t;
        l.e0 = t * p->tile_events;
        l.e1 = std::min(n_events, l.e0 + p->tile_events);
        l.h0 = h_event_offsets[l.e0];
        l.h1 = h_event_offsets[l.e1];
        if (l.h1 - l.h0 > p->max_hits || l.h1 < l.h0) { status = HOUGH_ERR_INVALID_ARG; l.tile = -1; break; }
        // the lane's pinned offset buffer is free: the previous H2D from it completed before `counted`
        for (int i = 0; i <= l.e1 - l.e0; ++i) l.h_off[i] = h_event_offsets[l.e0 + i] - l.h0;
        status = launch_part_a(p, l, h_hits_xy, threshold, assoc_dj, min_hits);
        if (status != HOUGH_OK) break;
        if (cudaEventRecord(l.counted, l.st) != cudaSuccess) { status = HOUGH_ERR_CUDA; break; }
    }
    // drain: tiles still in flight, in tile order
    if (status == HOUGH_OK) {
        std::vector<Lane*> order;
        for (Lane& l : p->lanes) if (l.tile >= 0) order.push_back(&l);
        std::sort(order.begin(), order.end(), [](const Lane* a, const Lane* b) { return a->tile < b->tile; });
        for (Lane* l : order) {
            status = finish(*l);
            if (status != HOUGH_OK) break;
        }
    }
    for (Lane& l : p->lanes) {
        if (cudaStreamSynchronize(l.st) != cudaSuccess && status == HOUGH_OK) {
            hough_set_last_cuda_error(cudaGetLastError(), "cudaStreamSynchronize");
            status = HOUGH_ERR_CUDA;
        }
        l.tile = -1;
    }
    return status;
}

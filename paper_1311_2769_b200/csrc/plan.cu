// plan.cu -- hough_plan_create / destroy, plan constants (D2), status strings.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <atomic>
#include <vector>
#include <algorithm>

#include "walk.cuh"

namespace {
thread_local char g_last_cuda[256] = "";
std::atomic<long long> g_launches{0};
}

void hough_count_launches(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
extern "C" int64_t hough_kernel_launches(void) { return (int64_t)g_launches.load(std::memory_order_relaxed); }

void hough_set_last_cuda_error(cudaError_t e, const char* what) {
    snprintf(g_last_cuda, sizeof(g_last_cuda), "%s: %s", what, cudaGetErrorString(e));
    if (getenv("HOUGH_VERBOSE")) fprintf(stderr, "[libhough_b200] CUDA error: %s\n", g_last_cuda);
    (void)cudaGetLastError();
}

extern "C" const char* hough_status_string(int status) {
    switch (status) {
        case HOUGH_OK: return "ok";
        case HOUGH_ERR_INVALID_ARG: return "invalid argument";
        case HOUGH_ERR_CUDA: return g_last_cuda[0] ? g_last_cuda : "CUDA error";
        case HOUGH_ERR_ALLOC: return "allocation failed";
        case HOUGH_ERR_UNSUPPORTED: return "unsupported configuration";
        case HOUGH_ERR_TOO_LARGE:
            return "size exceeds the fixed scratch of a no-allocation entry point (HOUGH_FIT_STATIC_MAX_CANDIDATES)";
        default: return "unknown status";
    }
}

extern "C" const char* hough_version(void) { return "libhough_b200 0.1 sm_100a"; }

static void plan_free(hough_plan* p) {
    if (!p) return;
    cudaFree(p->d_cs);
    cudaFree(p->d_d0t);
    cudaFree(p->d_peak_block_cnt);
    cudaFree(p->d_event_cnt);
    cudaFree(p->d_mask);
    cudaFree(p->d_word_rank);
    cudaFree(p->d_best_key);
    cudaFree(p->d_staged);
    cudaFree(p->d_stage_tmp);
    cudaFree(p->d_stage_cnt);
    cudaFree(p->d_slice);
    cudaFree(p->d_edge2);
    cudaFree(p->d_win);
    if (!p->assoc_tab_borrowed) cudaFree(p->d_assoc_tab);
    delete p;
}

extern "C" int hough_plan_create(const hough_binning* b, const hough_geometry* g, int32_t max_hits,
                                 int32_t max_events, hough_plan** out) {
    if (!b || !g || !out) return HOUGH_ERR_INVALID_ARG;
    if (b->n_phi <= 0 || b->n_phi % 4 != 0 || b->n_qpt <= 0 || b->n_d0 <= 0) return HOUGH_ERR_INVALID_ARG;
    if (!(b->qpt_max > b->qpt_min)) return HOUGH_ERR_INVALID_ARG;
    if (b->n_d0 > 1 && !(b->d0_max > b->d0_min)) return HOUGH_ERR_INVALID_ARG;
    if (b->accum_dtype != HOUGH_ACC_I32 && b->accum_dtype != HOUGH_ACC_U16) return HOUGH_ERR_INVALID_ARG;
    if (b->model != HOUGH_MODEL_HELIX && !(b->model == HOUGH_MODEL_LINE && b->n_d0 == 1)) return HOUGH_ERR_INVALID_ARG;
    if (max_hits <= 0 || max_events <= 0) return HOUGH_ERR_INVALID_ARG;
    if (g->n_layers < 0 || g->n_layers > 64 || (g->n_layers > 0 && !g->layer_radius_cm)) return HOUGH_ERR_INVALID_ARG;
    if (!(g->bz_tesla == g->bz_tesla)) return HOUGH_ERR_INVALID_ARG;
    const long long bins = (long long)b->n_phi * b->n_qpt * b->n_d0;
    if (bins > 0x7fffffffLL || b->n_qpt >= (1 << 24) || b->n_phi > (1 << 20) || b->n_d0 > (1 << 16))
        return HOUGH_ERR_UNSUPPORTED;

    hough_plan* p = new (std::nothrow) hough_plan();
    if (!p) return HOUGH_ERR_ALLOC;
    memset(p, 0, sizeof(*p));
    p->b = *b;
    p->bz = g->bz_tesla;
    p->max_hits = max_hits;
    p->max_events = max_events;
    p->n_layers = g->n_layers;
    for (int l = 0; l < g->n_layers; ++l) p->layer_r[l] = g->layer_radius_cm[l];
    const char* env = getenv("HOUGH_DEBUG_FULLSCAN");
    p->fullscan = (env && env[0] == '1') ? 1 : 0;
    env = getenv("HOUGH_DEBUG_EXACT_WALK");
    p->exact_walk = (env && env[0] == '1') ? 1 : 0;
    p->m_scale = 1.0f;
#ifdef HOUGH_CHECKS
    // self-check build only (never in libhough_b200.so): scale the fast path's error bound to probe its margin -- values
    // below 1 break bit-exactness on purpose (profiles/r2_walk.md)
    env = getenv("HOUGH_DEBUG_M_SCALE");
    if (env && atof(env) >= 0.0) p->m_scale = (float)atof(env);
#endif

    cudaError_t ce = cudaGetDevice(&p->device);
    if (ce == cudaSuccess) ce = cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, p->device);
    if (ce != cudaSuccess) { hough_set_last_cuda_error(ce, "cudaGetDevice"); delete p; return HOUGH_ERR_CUDA; }

    // ---- D2: constants, double -> fp32 ----
    const double kPi = 3.14159265358979323846;
    HoughConsts& c = p->c;
    c.n_phi = b->n_phi; c.n_qpt = b->n_qpt; c.n_d0 = b->n_d0;
    c.bins_per_event = (int32_t)bins;
    c.words_per_event = (int32_t)((bins + 31) / 32);
    c.is_u16 = b->accum_dtype == HOUGH_ACC_U16;
    c.model = b->model;
    c.A_f = (float)(0.5 * 0.00299792458 * (double)g->bz_tesla);
    c.qmin = b->qpt_min;
    c.inv_wq = (float)((double)b->n_qpt / ((double)b->qpt_max - (double)b->qpt_min));
    c.nq_f = (float)b->n_qpt;
    c.qpt_min = b->qpt_min;
    c.d0_min = b->d0_min;
    c.wq = (float)(((double)b->qpt_max - (double)b->qpt_min) / (double)b->n_qpt);
    c.wphi = (float)((2.0 * kPi) / (double)b->n_phi);
    c.wd = (float)(((double)b->d0_max - (double)b->d0_min) / (double)b->n_d0);
    c.two_pi_f = (float)(2.0 * kPi);
    {
        const double delta = 2.0 * kPi / (double)b->n_phi;
        c.kappa = (float)(4.0 * sin(delta) * sin(delta));
        c.sd2 = (float)(2.0 * sin(delta));
    }

    std::vector<float2> cs(b->n_phi);
    const int q = b->n_phi / 4;
    for (int i = 0; i < q; ++i) {
        const double th = ((double)i + 0.5) * (2.0 * kPi / (double)b->n_phi);
        cs[i].x = (float)cos(th);
        cs[i].y = (float)sin(th);
    }
    for (int i = 0; i + q < b->n_phi; ++i) {   // quarter-turn symmetry, exact
        cs[i + q].x = -cs[i].y;
        cs[i + q].y = cs[i].x;
    }
    std::vector<float4> d0t(b->n_d0);
    for (int k = 0; k < b->n_d0; ++k) {
        float d0c = 0.0f;
        if (b->n_d0 > 1)
            d0c = (float)((double)b->d0_min + ((double)k + 0.5) * ((double)b->d0_max - (double)b->d0_min) / (double)b->n_d0);
        d0t[k].x = d0c;
        d0t[k].y = 2.0f * d0c;
        d0t[k].z = d0c * d0c;
        d0t[k].w = 0.0f;
    }

    // ---- work sizing: radius classes, column windows, tile shape (results never depend on these) ----
    HoughWindows win;
    if (hough_build_windows(*b, g->bz_tesla, g->n_layers, g->layer_radius_cm, win) != HOUGH_OK) { delete p; return HOUGH_ERR_INVALID_ARG; }
    c.n_class = win.n_class;
    // one sector per phi0 column (clamped): fine enough for the candidate-centric association to read a candidate's
    // hits off the key-start table, and the vote walk is insensitive to the count above 32 (profiles/r1_final.md)
    c.n_sector = std::min(std::max(b->n_phi, HOUGH_SECTORS_MIN), HOUGH_SECTORS_MAX);
    // ... but the key-start table [max_events][n_class * n_sector + 1] is cleared and scanned by every staging call: halve
    // the sector count until the table is at most HOUGH_STAGE_TABLE_BYTES (a 1024-event plan with n_phi >= 1024 would
    // otherwise clear ~290 MB per call, 32x the 32-sector table).  Coarser sectors only make the candidate-centric
    // association read a few more hits per candidate.
    while (c.n_sector > HOUGH_SECTORS_MIN &&
           (long long)max_events * ((long long)c.n_class * c.n_sector + 1) * (long long)sizeof(int32_t) > HOUGH_STAGE_TABLE_BYTES)
        c.n_sector = std::max(c.n_sector / 2, HOUGH_SECTORS_MIN);
    { const char* es = getenv("HOUGH_SECTORS"); if (es && atoi(es) >= 1 && atoi(es) <= HOUGH_SECTORS_MAX) c.n_sector = atoi(es); }
    c.n_keys = c.n_class * c.n_sector;
    c.u_scale = (float)((double)b->n_phi / (2.0 * kPi));
    c.sector_scale = (float)((double)c.n_sector / (2.0 * kPi));
    std::vector<int2> winT((size_t)win.n_class * b->n_d0);
    for (size_t t = 0; t < winT.size(); ++t) {
        int lo_bits;
        memcpy(&lo_bits, &win.lo_off[t], 4);
        winT[t] = make_int2(lo_bits, win.steps[t] | (win.fwd_safe[t] ? (1 << 30) : 0));
    }
    p->event_max_steps = 0;
    // (the first and the open-ended last class span the whole circle by construction and hold no layer: left out)
    for (int cl = (win.n_class > 2 ? 1 : 0); cl < (win.n_class > 2 ? win.n_class - 1 : win.n_class); ++cl)
        p->event_max_steps = std::max(p->event_max_steps, std::min(win.steps[(size_t)cl * b->n_d0], (int)b->n_phi));
    // packed 16-bit tiles are exact whenever no bin can exceed 65535: the U16 precondition, or at most 65535
    // hits per call (a hit casts at most one vote per (phi0, d0) column, D3)
    p->tile32 = (b->accum_dtype == HOUGH_ACC_I32 && max_hits > 65535) ? 1 : 0;
#ifdef HOUGH_CHECKS
    { const char* et = getenv("HOUGH_FORCE_TILE32"); if (et && et[0] == '1') p->tile32 = 1; }   // layout experiments, checks build only
#endif
    {
        // walk.cuh "Tile layout": a row (32-bit bins) or a row of column PAIRS (16-bit bins) has `stride` words.
        // Largest even column count whose whole shared-memory block lets 3 CTAs share an SM (228 KB, 1 KB reserved per
        // CTA); rows too wide for that get one big tile per SM.
        const int stride = walk_row_stride(b->n_qpt);
        p->tile_stride_words = stride;
        auto fit = [&](size_t budget) {
            int lo = 0, hi = b->n_phi / 2;                                // pairs of columns
            while (lo < hi) {
                const int mid = (lo + hi + 1) / 2;
                if (walk_smem_bytes(2 * mid, stride, p->tile32 != 0, win.n_class, 2 * mid == b->n_phi) <= budget) lo = mid; else hi = mid - 1;
            }
            return 2 * lo;
        };
        int cols = fit((size_t)(233472 / 3 - 1024 - 64));
        if (cols < 8) cols = fit((size_t)(200 * 1024));
        p->tile_max_cols = cols;                                          // 0: no tiled path (fullscan fallback)
    }

    p->peak_blocks_per_event = (int32_t)((bins + PEAK_BLOCK_BINS - 1) / PEAK_BLOCK_BINS);
    const size_t n_words = (size_t)max_events * c.words_per_event;

    bool ok = true;
    auto A = [&](void** ptr, size_t bytes) {
        if (!ok) return;
        if (cudaMalloc(ptr, bytes ? bytes : 4) != cudaSuccess) { ok = false; (void)cudaGetLastError(); }
    };
    A((void**)&p->d_cs, sizeof(float2) * ((size_t)b->n_phi + 2));      // two pad entries in front: c.cs[-1] = column n_phi - 1
    A((void**)&p->d_d0t, sizeof(float4) * b->n_d0);
    A((void**)&p->d_peak_block_cnt, sizeof(int32_t) * (size_t)max_events * p->peak_blocks_per_event);
    A((void**)&p->d_event_cnt, sizeof(int32_t) * ((size_t)max_events + 1));
    A((void**)&p->d_mask, sizeof(uint32_t) * n_words);
    A((void**)&p->d_word_rank, sizeof(int32_t) * n_words);
    A((void**)&p->d_best_key, sizeof(unsigned long long) * (size_t)max_hits);
    A((void**)&p->d_staged, sizeof(float4) * (size_t)max_hits);
    A((void**)&p->d_stage_tmp, sizeof(int2) * (size_t)max_hits);
    A((void**)&p->d_stage_cnt, sizeof(int32_t) * (size_t)max_events * ((size_t)c.n_keys + 1));
    // tiles per call: walk_shape() never uses more slabs than ceil(n_phi / 32) or than the budget needs
    {
        const long long slabs_budget = p->tile_max_cols >= 1 ? (b->n_phi + p->tile_max_cols - 1) / p->tile_max_cols : 1;
        const long long slabs_max = std::max<long long>(2 * slabs_budget, (b->n_phi + 31) / 32 * 2);
        p->slice_len = (size_t)max_events * (size_t)b->n_d0 * (size_t)slabs_max;
    }
    A((void**)&p->d_slice, sizeof(int2) * p->slice_len);
    A((void**)&p->d_edge2, sizeof(float) * win.n_class);
    A((void**)&p->d_win, sizeof(int2) * winT.size());
    if (!ok) { plan_free(p); return HOUGH_ERR_ALLOC; }
    cs.insert(cs.begin(), 2, cs[b->n_phi - 1]);
    if (cudaMemcpy(p->d_cs, cs.data(), sizeof(float2) * ((size_t)b->n_phi + 2), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(p->d_edge2, win.edge2.data(), sizeof(float) * win.n_class, cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(p->d_win, winT.data(), sizeof(int2) * winT.size(), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(p->d_d0t, d0t.data(), sizeof(float4) * b->n_d0, cudaMemcpyHostToDevice) != cudaSuccess) {
        hough_set_last_cuda_error(cudaGetLastError(), "table upload");
        plan_free(p);
        return HOUGH_ERR_CUDA;
    }
    c.cs = p->d_cs + 2;                       // 16-byte aligned; c.cs[-1] is the wrap-around column (walk.cuh wrec_init)
    c.d0t = p->d_d0t;
    c.edge2 = p->d_edge2;
    c.win = p->d_win;
    *out = p;
    return HOUGH_OK;
}

extern "C" int hough_plan_destroy(hough_plan* p) {
    if (!p) return HOUGH_ERR_INVALID_ARG;
    plan_free(p);
    return HOUGH_OK;
}

extern "C" size_t hough_accum_bytes(const hough_plan* p, int32_t n_events) {
    if (!p || n_events < 0) return 0;
    return (size_t)n_events * (size_t)p->c.bins_per_event * (p->c.is_u16 ? 2 : 4);
}

extern "C" int hough_plan_set_option(hough_plan* p, const char* key, int32_t value) {
    if (!p || !key) return HOUGH_ERR_INVALID_ARG;
    if (strcmp(key, "fullscan") == 0) { p->fullscan = value ? 1 : 0; return HOUGH_OK; }
    if (strcmp(key, "peaks_tiled") == 0) { p->peaks_tiled = value ? 1 : 0; return HOUGH_OK; }
    if (strcmp(key, "peaks_regs") == 0) { p->peaks_regs = value ? 1 : 0; return HOUGH_OK; }
    if (strcmp(key, "peaks_scalar") == 0) { p->peaks_scalar = value ? 1 : 0; return HOUGH_OK; }
    if (strcmp(key, "assign_candidates") == 0) {
        p->assign_candidates = value ? 1 : 0;
        if (value && !p->d_assoc_tab && p->tile_max_cols >= 1) { p->assoc_tab_tried = 1; return hough_build_assoc_table(p); }   // built once, on first use
        return HOUGH_OK;
    }
    if (strcmp(key, "event_cluster") == 0) { p->event_cluster = value ? 1 : 0; return HOUGH_OK; }
    if (strcmp(key, "event_general") == 0) { p->event_general = value ? 1 : 0; return HOUGH_OK; }
    if (strcmp(key, "reassign_walk") == 0) { p->reassign_walk = value ? 1 : 0; return HOUGH_OK; }
    if (strcmp(key, "prepare_reassign") == 0) return value ? hough_prepare_reassign(p) : HOUGH_OK;
    if (strcmp(key, "exact_walk") == 0) { p->exact_walk = value ? 1 : 0; return HOUGH_OK; }
    if (strcmp(key, "reuse_staging") == 0) { p->reuse_staging = value ? 1 : 0; p->staged_hits = nullptr; return HOUGH_OK; }
    return HOUGH_ERR_INVALID_ARG;
}

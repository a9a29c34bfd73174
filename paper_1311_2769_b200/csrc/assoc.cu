// assoc.cu -- A5, candidate-centric hit association ("further computations ... to confirm the existence of the
// track"; D8).  Plan option "assign_candidates" (off by default: measured slower than the column walk: 4.6 vs 2.2 ms per 256-event call, profiles/r2_walk.md).
//
// D8 asks, for every hit, for the best candidate among those whose column (i, k) the hit votes in within assoc_dj bins
// of the candidate's bin.  Candidates are few compared with vote positions (config 3: 2.6e4 candidates against 6.4e6
// vote positions per event), so the work is turned round: for every candidate (k, i, j) and every radius class that
// holds hits, the hits that can land in bins [j - dj, j + dj] of column (i, k) lie in one short azimuth interval.
//   * assoc table (plan creation, double precision, built on the device): for (class, d0 slice, bin EDGE e) the hull,
//     over the class's radius interval, of the azimuth offset (hit azimuth - column centre, in column units) at which
//     the D3 function t equals e.  t is monotone in the azimuth for fixed (r, column), so the hits of bins
//     [j - dj, j + dj] lie between the entries of edges j - dj and j + dj + 1.  Margins make the interval a superset
//     (work sizing only: S19); what decides is the exact D3 sequence run on every hit of the interval.
//   * the staged hits are sorted by (event, class, fine phi sector) (stage.cu), so the interval is a contiguous range of
//     staged positions read off the key-start table.
//   * lane = candidate (32 consecutive records: same slice, neighbouring columns); loop over the event's non-empty
//     classes; the D8 key (votes, -|dj|, -candidate index) is folded into a per-hit best key held in shared memory
//     (one CTA works on one event) and merged into the global array with one atomicMax per touched hit at the end.
//     Events with more hits than the shared-memory array holds fold straight into global memory (look first, then
//     atomicMax).
#include <algorithm>
#include <cmath>

#include "walk.cuh"

namespace {

// ---- assoc table -----------------------------------------------------------------------------------------------------
// hull of S(r) = a / r - b r over r in [ra, rb], ra > 0
__device__ void hull_S_dev(double a, double b, double ra, double rb, double& smin, double& smax) {
    const double s0 = a / ra - b * ra, s1 = a / rb - b * rb;
    smin = fmin(s0, s1);
    smax = fmax(s0, s1);
    if (b != 0.0 && -a / b > 0.0) {                      // interior extremum at r* = sqrt(-a / b)
        const double rs = sqrt(-a / b);
        if (rs > ra && rs < rb) {
            const double ss = a / rs - b * rs;
            smin = fmin(smin, ss);
            smax = fmax(smax, ss);
        }
    }
}

// entry (class cl, slice k, edge e) = {lo, hi}: every hit of the class whose D3 value t at a column equals e (up to the
// roundings of the fp32 sequence, covered by eps_q and the s-margins) has  lo <= u_hit - column <= hi.  {-n_phi, n_phi}
// means "no bound" (the candidate then scans the whole class).
__global__ void __launch_bounds__(256) assoc_table_kernel(HoughConsts c, double A, double qmin, double qmax, float2* __restrict__ tab) {
    const int nq1 = c.n_qpt + 1;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long n = (long long)c.n_class * c.n_d0 * nq1;
    if (t >= n) return;
    const int e = (int)(t % nq1);
    const int k = (int)((t / nq1) % c.n_d0);
    const int cl = (int)(t / ((long long)nq1 * c.n_d0));
    const float full = (float)c.n_phi;
    float2 out = make_float2(-full, full);
    const double cols_per_rad = (double)c.n_phi / 6.283185307179586476925;
    const bool open = cl == c.n_class - 1;
    const double ra = sqrt((double)c.edge2[cl]) * (1.0 - 1.0e-6);
    const double rb = open ? 0.0 : sqrt((double)c.edge2[cl + 1]) * (1.0 + 1.0e-6);
    const double eps = 1.0e-5 * (fabs(qmin) + fabs(qmax));
    const double qe = qmin + (double)e * (qmax - qmin) / (double)c.n_qpt;
    double s_lo = 0.0, s_hi = 0.0;
    bool ok = !open && ra > 0.0 && rb > ra;
    if (ok && c.model != 0) {
        // D3L: t = (w - qmin) inv_w with w = r sin(phi - phi0): s = q_e / r
        const double a0 = (qe - eps), a1 = (qe + eps);
        s_lo = fmin(fmin(a0 / ra, a0 / rb), fmin(a1 / ra, a1 / rb));
        s_hi = fmax(fmax(a0 / ra, a0 / rb), fmax(a1 / ra, a1 / rb));
    } else if (ok) {
        ok = A > 0.0;
        const double d0 = (double)c.d0t[k].x;
        s_lo = 1.0e30; s_hi = -1.0e30;
        for (int sgn = -1; sgn <= 1 && ok; sgn += 2) {
            const double q = qe + sgn * eps;
            const double cq = 1.0 - 2.0 * q * A * d0;
            if (!(cq > 1.0e-3)) { ok = false; break; }
            double lo, hi;
            hull_S_dev(d0 * (1.0 - q * A * d0) / cq, q * A / cq, ra, rb, lo, hi);      // sin(phi - phi0) = S(q; r)
            s_lo = fmin(s_lo, lo);
            s_hi = fmax(s_hi, hi);
        }
    }
    if (ok && isfinite(s_lo) && isfinite(s_hi)) {
        s_lo -= 1.0e-5 + 1.0e-6 * fabs(s_lo);
        s_hi += 1.0e-5 + 1.0e-6 * fabs(s_hi);
        const double d_lo = asin(fmax(fmin(s_lo, 1.0), -1.0)) * cols_per_rad;
        const double d_hi = asin(fmax(fmin(s_hi, 1.0), -1.0)) * cols_per_rad;
        out.x = __double2float_rd(d_lo);
        out.y = __double2float_ru(d_hi);
    }
    tab[t] = out;
}

// ---- association -----------------------------------------------------------------------------------------------------
struct AssocArgs {
    const float4* staged;            // [n_hits] staged hits {x, y, u, bits(original index)}
    const int32_t* off;              // [n_events + 1]
    const int32_t* key_start;        // [n_events][n_keys + 1]
    const hough_candidate* cands;
    const int32_t* cand_off;         // [n_events + 1]
    const float2* tab;               // assoc table
    unsigned long long* best_key;    // [n_hits] by original hit index
    const uint8_t* keep;             // optional [capacity]: only candidates with keep != 0 take part (D12)
    int capacity, assoc_dj, parts;
    int smem_hits;                   // entries of the shared best-key array (events with more hits fold into global memory)
    float margin_cols, sec_per_col;
};

__device__ __forceinline__ unsigned long long assoc_key(int votes, int adj, int index) {
    return ((unsigned long long)(unsigned)votes << 40) | ((unsigned long long)(255 - adj) << 32) |
           (unsigned long long)(0xFFFFFFFFu - (unsigned)index);
}

constexpr int ASSOC_THREADS = 384;                    // 12 warps; 3 CTAs per SM next to a 73 KB best-key array
constexpr int ASSOC_WARPS = ASSOC_THREADS / 32;
constexpr int ASSOC_PASSES = 3;                       // candidates are taken in passes of descending votes (see below)
constexpr int ASSOC_HIST = 256;

// Best key of staged hit `pos` of the event: shared array, or the global array for events too large for it.
template <bool SMEM>
__device__ __forceinline__ unsigned long long assoc_best(const unsigned long long* s_best, const unsigned long long* g_best, int pos) {
    if (SMEM) return *reinterpret_cast<const volatile unsigned long long*>(s_best + pos);
    return __ldcg(g_best + pos);
}

// One warp, 32 candidates (lane = candidate `ci`, or -1): for every non-empty class, walk the staged hits of the
// candidate's azimuth interval.  A hit whose best key already beats the best key this candidate could give it
// (|dj| = 0) is skipped after one load and one compare; the others get the exact D3 sequence.  The evaluations are
// deferred to warp-synchronous rounds so that lanes still scanning do not drag the whole warp through them.
template <bool SMEM>
__device__ __forceinline__ void assoc_group(const HoughConsts& c, const AssocArgs& a, const int32_t* __restrict__ ks, int ev_begin,
                                            const short* s_cls, int ncl, unsigned long long* s_best, unsigned long long* g_best,
                                            int ci) {
    const bool valid = ci >= 0;
    const int NS = c.n_sector, nq = c.n_qpt, nq1 = nq + 1, dj = a.assoc_dj;
    const int4 q = valid ? __ldg(reinterpret_cast<const int4*>(a.cands + ci)) : make_int4(0, 0, 0, 0);      // event, k, i, j
    const int votes = valid ? __ldg(&a.cands[ci].votes) : 0;
    const float2 cs = __ldg(c.cs + q.z);
    const float4 d = __ldg(c.d0t + q.y);
    const int e_lo = max(q.w - dj, 0), e_hi = min(q.w + dj + 1, nq);
    const float col = (float)q.z;
    const unsigned long long ub_key = assoc_key(votes, 0, ci);          // the best this candidate can offer any hit
    const bool line = c.model != 0;
    for (int s = 0; s < ncl; ++s) {
        const int cl = s_cls[s];
        const float2* tb = a.tab + ((size_t)cl * c.n_d0 + q.y) * nq1;
        const float2 ta = __ldg(tb + e_lo), tz = __ldg(tb + e_hi);
        const float ua = col + fminf(ta.x, tz.x) - a.margin_cols;
        const float ub = col + fmaxf(ta.y, tz.y) + a.margin_cols;
        // staged positions of the sectors that meet [ua, ub] (cyclic); the whole class when the interval is unbounded
        const float fa = floorf((ua + 0.5f) * a.sec_per_col - 1.0e-3f);
        const float fb = floorf((ub + 0.5f) * a.sec_per_col + 1.0e-3f);
        const int base = cl * NS;
        int p0, n0, p1 = 0, n1 = 0;
        const float nsf = fb - fa + 1.0f;
        if (!(nsf < (float)NS)) {
            p0 = __ldg(ks + base);
            n0 = __ldg(ks + base + NS) - p0;
        } else {
            const int ns = (int)nsf;
            int sa = (int)fa % NS;
            if (sa < 0) sa += NS;
            p0 = __ldg(ks + base + sa);
            if (sa + ns <= NS) {
                n0 = __ldg(ks + base + sa + ns) - p0;
            } else {
                n0 = __ldg(ks + base + NS) - p0;
                p1 = __ldg(ks + base);
                n1 = __ldg(ks + base + sa + ns - NS) - p1;
            }
        }
        const int n = valid ? n0 + n1 : 0;
        const int shift = p1 - p0 - n0;                                  // position of logical index t >= n0: p0 + t + shift
        int t = 0;
        for (;;) {
            int found = -1;
            while (t < n) {
                const int pos = p0 + t + (t >= n0 ? shift : 0);
                ++t;
                if (ub_key > assoc_best<SMEM>(s_best, g_best, SMEM ? pos : ev_begin + pos)) { found = pos; break; }
            }
            if (!__any_sync(0xffffffffu, found >= 0)) break;
            if (found >= 0) {
                const float4 hv = __ldg(a.staged + ev_begin + found);
                const int jh = d3_exact_bin(hv.x, hv.y, d3_r2(hv.x, hv.y), cs.x, cs.y, d.x, d.y, d.z, c.A_f, c.qmin, c.inv_wq, c.nq_f,
                                            line);
                const int adj = abs(jh - q.w);
                if (jh >= 0 && adj <= dj) {
                    const unsigned long long key = assoc_key(votes, adj, ci);
                    unsigned long long* bp = SMEM ? s_best + found : g_best + ev_begin + found;
                    if (key > assoc_best<SMEM>(s_best, g_best, SMEM ? found : ev_begin + found)) atomicMax(bp, key);
                }
            }
        }
    }
}

// Grid = n_events x parts; a CTA takes a contiguous chunk of one event's candidate list.  Pass structure: a vote
// histogram of the chunk gives two vote levels; pass 0 takes the candidates at or above the upper level (the top few
// per cent), pass 1 those down to the lower level, pass 2 the rest, with a CTA barrier in between -- by the time the
// many low-vote (combinatorial) candidates are looked at, most hits already hold a better key and are skipped.  The
// order changes how much work is done, never the result (max is order-free).  Inside a pass every warp compacts the
// selected candidates of its sub-range 32 at a time (ballot), keeping the list order: neighbouring lanes share a slice
// and neighbouring columns, so table rows and staged hits are read with locality.
// Best keys live by STAGED position (shared memory: inside the event; global fallback: inside the call) and are
// translated to original hit indices when they are merged / decoded.
template <bool SMEM>
__global__ void __launch_bounds__(ASSOC_THREADS, SMEM ? 3 : 2) assoc_cand_kernel(HoughConsts c, AssocArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ int s_ncl;
    __shared__ int s_level[2];
    __shared__ int s_hist[ASSOC_HIST];
    __shared__ short s_cls[HOUGH_MAX_CLASSES + 1];
    __shared__ int s_q[ASSOC_WARPS][64];
    unsigned long long* s_best = reinterpret_cast<unsigned long long*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int e = blockIdx.x / a.parts, part = blockIdx.x % a.parts;
    const int first = min(__ldg(a.cand_off + e), a.capacity), end = min(__ldg(a.cand_off + e + 1), a.capacity);
    const int n_c = end - first;
    if (n_c <= 0) return;
    const int chunk = (((n_c + a.parts - 1) / a.parts) + 31) & ~31;
    const int c_begin = first + part * chunk, c_end = min(c_begin + chunk, end);
    if (c_begin >= c_end) return;
    const int ev_begin = __ldg(a.off + e);
    const int ev_hits = __ldg(a.off + e + 1) - ev_begin;
    if (ev_hits <= 0) return;
    if (SMEM != (ev_hits <= a.smem_hits)) return;          // the other instantiation's launch takes this event
    const int NS = c.n_sector, nc = c.n_class;
    const int32_t* ks = a.key_start + (size_t)e * (c.n_keys + 1);
    if (tid == 0) s_ncl = 0;
    for (int x = tid; x < ASSOC_HIST; x += ASSOC_THREADS) s_hist[x] = 0;
    __syncthreads();
    for (int cl = tid; cl < nc; cl += ASSOC_THREADS)
        if (__ldg(ks + (cl + 1) * NS) > __ldg(ks + cl * NS)) s_cls[atomicAdd(&s_ncl, 1)] = (short)cl;
    if (SMEM)
        for (int h = tid; h < ev_hits; h += ASSOC_THREADS) s_best[h] = 0ull;
    for (int ci = c_begin + tid; ci < c_end; ci += ASSOC_THREADS)
        if (!a.keep || __ldg(a.keep + ci)) atomicAdd(&s_hist[min(max(__ldg(&a.cands[ci].votes), 0), ASSOC_HIST - 1)], 1);
    __syncthreads();
    if (tid == 0) {                                        // vote levels: top ~1/16 and top ~1/3 of the chunk
        int total = 0;
        for (int v = 0; v < ASSOC_HIST; ++v) total += s_hist[v];
        int acc = 0, l0 = ASSOC_HIST, l1 = ASSOC_HIST;
        for (int v = ASSOC_HIST - 1; v >= 0; --v) {
            acc += s_hist[v];
            if (l0 == ASSOC_HIST && acc * 16 >= total) l0 = v;
            if (l1 == ASSOC_HIST && acc * 3 >= total) { l1 = v; break; }
        }
        s_level[0] = l0;
        s_level[1] = min(l1, l0);
    }
    __syncthreads();
    const int ncl = s_ncl;
    // the warp's sub-range of the chunk (whole groups of 32)
    const int groups = (c_end - c_begin + 31) >> 5;
    const int g_per_warp = (groups + ASSOC_WARPS - 1) / ASSOC_WARPS;
    const int w_begin = c_begin + warp * g_per_warp * 32, w_end = min(w_begin + g_per_warp * 32, c_end);
    int* wq = s_q[warp];
    unsigned long long* g_best = a.best_key;
    for (int pass = 0; pass < ASSOC_PASSES; ++pass) {
        const int v_hi = pass == 0 ? 0x7fffffff : s_level[pass - 1];      // votes in [v_lo, v_hi), clamped like the histogram
        const int v_lo = pass == ASSOC_PASSES - 1 ? -1 : s_level[pass];
        int qn = 0;
        for (int g = w_begin; g < w_end; g += 32) {
            const int ci = g + lane;
            bool sel = false;
            if (ci < w_end && (!a.keep || __ldg(a.keep + ci))) {
                const int v = min(max(__ldg(&a.cands[ci].votes), 0), ASSOC_HIST - 1);
                sel = v >= v_lo && v < v_hi;
            }
            const unsigned bal = __ballot_sync(0xffffffffu, sel);
            if (sel) wq[qn + __popc(bal & ((1u << lane) - 1u))] = ci;
            qn += __popc(bal);
            __syncwarp();
            if (qn >= 32) {
                assoc_group<SMEM>(c, a, ks, ev_begin, s_cls, ncl, s_best, g_best, wq[lane]);
                __syncwarp();
                if (lane < qn - 32) wq[lane] = wq[32 + lane];
                qn -= 32;
                __syncwarp();
            }
        }
        if (qn > 0) assoc_group<SMEM>(c, a, ks, ev_begin, s_cls, ncl, s_best, g_best, lane < qn ? wq[lane] : -1);
        __syncthreads();
    }
    if (!SMEM) return;
    for (int h = tid; h < ev_hits; h += ASSOC_THREADS) {
        const unsigned long long key = s_best[h];
        if (key) atomicMax(g_best + ev_begin + h, key);
    }
}

// ---- few candidates (D12 round: only the survivors of duplicate removal take part) -----------------------------------
// With a keep filter a CTA's chunk holds a handful of participating candidates (config 3: 188 of 25 600 per event), far
// too few to fill warps with lane = candidate.  Here the kept candidates of the chunk are compacted into shared memory
// and the (candidate, class) ITEMS are dealt to the threads, so a few hundred candidates still give thousands of
// independent items.  Keys are folded straight into the global best-key array (look first, then atomicMax).
constexpr int ASSOC_KEPT_THREADS = 256;
constexpr int ASSOC_KEPT_CHUNK = 4096;                // candidates examined per round: bounds the shared list

__global__ void __launch_bounds__(ASSOC_KEPT_THREADS) assoc_kept_kernel(HoughConsts c, AssocArgs a) {
    __shared__ int s_list[ASSOC_KEPT_CHUNK];
    __shared__ int s_n, s_ncl;
    __shared__ short s_cls[HOUGH_MAX_CLASSES + 1];
    const int tid = threadIdx.x;
    const int e = blockIdx.x / a.parts, part = blockIdx.x % a.parts;
    const int first = min(__ldg(a.cand_off + e), a.capacity), end = min(__ldg(a.cand_off + e + 1), a.capacity);
    const int n_c = end - first;
    if (n_c <= 0) return;
    const int chunk = (n_c + a.parts - 1) / a.parts;
    const int c_begin = first + part * chunk, c_end = min(c_begin + chunk, end);
    if (c_begin >= c_end) return;
    const int ev_begin = __ldg(a.off + e);
    const int ev_hits = __ldg(a.off + e + 1) - ev_begin;
    if (ev_hits <= 0) return;
    const int NS = c.n_sector, nc = c.n_class, nq = c.n_qpt, nq1 = nq + 1, dj = a.assoc_dj;
    const int32_t* ks = a.key_start + (size_t)e * (c.n_keys + 1);
    const bool line = c.model != 0;
    if (tid == 0) s_ncl = 0;
    __syncthreads();
    for (int cl = tid; cl < nc; cl += ASSOC_KEPT_THREADS)
        if (__ldg(ks + (cl + 1) * NS) > __ldg(ks + cl * NS)) s_cls[atomicAdd(&s_ncl, 1)] = (short)cl;
    for (int r0 = c_begin; r0 < c_end; r0 += ASSOC_KEPT_CHUNK) {
        __syncthreads();
        if (tid == 0) s_n = 0;
        __syncthreads();
        const int r1 = min(r0 + ASSOC_KEPT_CHUNK, c_end);
        for (int ci = r0 + tid; ci < r1; ci += ASSOC_KEPT_THREADS)
            if (!a.keep || __ldg(a.keep + ci)) s_list[atomicAdd(&s_n, 1)] = ci;
        __syncthreads();
        const int ncl = s_ncl, items = s_n * ncl;
        for (int item = tid; item < items; item += ASSOC_KEPT_THREADS) {
            const int ci = s_list[item / ncl], cl = s_cls[item % ncl];
            const int4 q = __ldg(reinterpret_cast<const int4*>(a.cands + ci));          // event, k, i, j
            const int votes = __ldg(&a.cands[ci].votes);
            const float2 cs = __ldg(c.cs + q.z);
            const float4 d = __ldg(c.d0t + q.y);
            const int e_lo = max(q.w - dj, 0), e_hi = min(q.w + dj + 1, nq);
            const float2* tb = a.tab + ((size_t)cl * c.n_d0 + q.y) * nq1;
            const float2 ta = __ldg(tb + e_lo), tz = __ldg(tb + e_hi);
            const float col = (float)q.z;
            const float ua = col + fminf(ta.x, tz.x) - a.margin_cols;
            const float ub = col + fmaxf(ta.y, tz.y) + a.margin_cols;
            const float fa = floorf((ua + 0.5f) * a.sec_per_col - 1.0e-3f);
            const float fb = floorf((ub + 0.5f) * a.sec_per_col + 1.0e-3f);
            const int base = cl * NS;
            int p0, n0, p1 = 0, n1 = 0;
            const float nsf = fb - fa + 1.0f;
            if (!(nsf < (float)NS)) {
                p0 = __ldg(ks + base);
                n0 = __ldg(ks + base + NS) - p0;
            } else {
                const int ns = (int)nsf;
                int sa = (int)fa % NS;
                if (sa < 0) sa += NS;
                p0 = __ldg(ks + base + sa);
                if (sa + ns <= NS) {
                    n0 = __ldg(ks + base + sa + ns) - p0;
                } else {
                    n0 = __ldg(ks + base + NS) - p0;
                    p1 = __ldg(ks + base);
                    n1 = __ldg(ks + base + sa + ns - NS) - p1;
                }
            }
            const unsigned long long ub_key = assoc_key(votes, 0, ci);      // the best this candidate can offer any hit
            for (int t = 0; t < n0 + n1; ++t) {
                const int pos = t < n0 ? p0 + t : p1 + (t - n0);
                unsigned long long* bp = a.best_key + ev_begin + pos;
                if (!(ub_key > __ldcg(bp))) continue;
                const float4 hv = __ldg(a.staged + ev_begin + pos);
                const int jh = d3_exact_bin(hv.x, hv.y, d3_r2(hv.x, hv.y), cs.x, cs.y, d.x, d.y, d.z, c.A_f, c.qmin, c.inv_wq, c.nq_f,
                                            line);
                const int adj = abs(jh - q.w);
                if (jh >= 0 && adj <= dj) {
                    const unsigned long long key = assoc_key(votes, adj, ci);
                    if (key > __ldcg(bp)) atomicMax(bp, key);
                }
            }
        }
    }
}

// best key by staged position -> hit_to_cand by original hit index, and the per-candidate hit counts
// ORPHANS (D12 re-assignment round): only hits still at -1 take the new key; the others and their counts stay.
template <bool ORPHANS>
__global__ void __launch_bounds__(256) assoc_decode_kernel(const unsigned long long* __restrict__ best_key, const float4* __restrict__ staged,
                                                           int n_hits, int32_t* __restrict__ hit_to_cand, int32_t* __restrict__ cand_nhits) {
    const int pos = blockIdx.x * blockDim.x + threadIdx.x;
    if (pos >= n_hits) return;
    const unsigned long long key = best_key[pos];
    const int h = __float_as_int(__ldg(staged + pos).w);
    if (ORPHANS && (!key || hit_to_cand[h] >= 0)) return;
    int ci = -1;
    if (key) {
        ci = (int)(0xFFFFFFFFu - (unsigned)(key & 0xFFFFFFFFull));
        atomicAdd(cand_nhits + ci, 1);
    }
    hit_to_cand[h] = ci;
}

}  // namespace

// Build the plan's assoc table (device, double precision).  Leaves p->d_assoc_tab null when it would not fit the
// budget (the association then takes the column walk).
int hough_build_assoc_table(hough_plan* p) {
    p->d_assoc_tab = nullptr;
    const long long n = (long long)p->c.n_class * p->c.n_d0 * (p->c.n_qpt + 1);
    if (n * (long long)sizeof(float2) > (96LL << 20)) return HOUGH_OK;
    float2* tab = nullptr;
    if (cudaMalloc((void**)&tab, (size_t)n * sizeof(float2)) != cudaSuccess) { (void)cudaGetLastError(); return HOUGH_ERR_ALLOC; }
    const double A = (double)p->c.A_f;
    assoc_table_kernel<<<(unsigned)((n + 255) / 256), 256>>>(p->c, A, (double)p->b.qpt_min, (double)p->b.qpt_max, tab);
    cudaError_t ce = cudaGetLastError();
    if (ce == cudaSuccess) ce = cudaDeviceSynchronize();
    if (ce != cudaSuccess) { hough_set_last_cuda_error(ce, "assoc_table_kernel"); cudaFree(tab); return HOUGH_ERR_CUDA; }
    hough_count_launches(1);
    p->d_assoc_tab = tab;
    return HOUGH_OK;
}

int hough_prepare_reassign(hough_plan* p) {
    if (p->d_assoc_tab || p->assoc_tab_tried || p->fullscan || p->tile_max_cols < 1) return HOUGH_OK;
    p->assoc_tab_tried = 1;
    if (hough_build_assoc_table(p) != HOUGH_OK) p->d_assoc_tab = nullptr;      // no table: the D12 round re-walks the columns
    return HOUGH_OK;
}

// Candidate-centric association of a staged call: folds the D8 keys into p->d_best_key (zeroed by the caller, indexed by
// STAGED position) and decodes them into d_hit_to_cand / d_cand_nhits.
int hough_assoc_candidates(hough_plan* p, const int32_t* d_event_offsets, int32_t n_hits, int32_t n_events,
                           const hough_candidate* d_cands, const int32_t* d_cand_offsets, int32_t capacity, int32_t assoc_dj,
                           int32_t* d_hit_to_cand, int32_t* d_cand_nhits, cudaStream_t st, const uint8_t* d_keep_filter) {
    AssocArgs a{};
    a.keep = d_keep_filter;
    a.staged = p->d_staged;
    a.off = d_event_offsets;
    a.key_start = p->d_stage_cnt;
    a.cands = d_cands;
    a.cand_off = d_cand_offsets;
    a.tab = p->d_assoc_tab;
    a.best_key = p->d_best_key;
    a.capacity = capacity;
    a.assoc_dj = assoc_dj;
    // about two waves of CTAs (3 per SM); more parts balance better but weaken the skipping and repeat the merge
    long long parts = (2LL * 3 * p->sm_count + n_events / 2) / n_events;
    if (parts < 1) parts = 1;
    if (parts > 1024) parts = 1024;
    a.parts = (int)parts;
    // shared best-key array: sized from the plan's average event (3 CTAs per SM when it fits 72 KB); events that do
    // not fit fold into global memory (second instantiation, launched when the plan allows such events)
    const long long per_event = ((long long)p->max_hits + p->max_events - 1) / p->max_events;
    const long long want_hits = per_event + per_event / 8 + 64;
    const int smem_hits = want_hits <= 9000 ? 9000 : (want_hits <= 13800 ? 13800 : (want_hits <= 28000 ? 28000 : 0));   // 3, 2, 1 CTAs per SM
    a.smem_hits = smem_hits;
    a.margin_cols = 0.02f + 4.0e-6f * (float)p->c.n_phi;
    a.sec_per_col = (float)((double)p->c.n_sector / (double)p->c.n_phi);
    const size_t smem = (size_t)smem_hits * sizeof(unsigned long long);
    if (smem > (size_t)p->assoc_smem_configured) {
        HOUGH_CUDA_TRY(cudaFuncSetAttribute(assoc_cand_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        p->assoc_smem_configured = (int)smem;
    }
    const long long grid = (long long)n_events * a.parts;
    if (grid > 0x7fffffffLL) return HOUGH_ERR_UNSUPPORTED;
    int launches = 1;
    if (d_keep_filter) {
        // D12 round: few survivors per event -> (candidate, class) items dealt to threads, keys straight into global memory
        long long kp = (4LL * p->sm_count + n_events - 1) / n_events;
        a.parts = (int)std::min<long long>(std::max<long long>(kp, 1), 64);
        assoc_kept_kernel<<<(unsigned)((long long)n_events * a.parts), ASSOC_KEPT_THREADS, 0, st>>>(p->c, a);
        HOUGH_CUDA_TRY(cudaGetLastError());
        assoc_decode_kernel<true><<<(n_hits + 255) / 256, 256, 0, st>>>(p->d_best_key, p->d_staged, n_hits, d_hit_to_cand, d_cand_nhits);
        HOUGH_CUDA_TRY(cudaGetLastError());
        hough_count_launches(2);
        return HOUGH_OK;
    }
    if (smem_hits > 0) {
        assoc_cand_kernel<true><<<(unsigned)grid, ASSOC_THREADS, smem, st>>>(p->c, a);
        HOUGH_CUDA_TRY(cudaGetLastError());
        ++launches;
    }
    if (p->max_hits > smem_hits) {                           // an event of this plan may exceed the shared array
        assoc_cand_kernel<false><<<(unsigned)grid, ASSOC_THREADS, 0, st>>>(p->c, a);
        HOUGH_CUDA_TRY(cudaGetLastError());
        ++launches;
    }
    assoc_decode_kernel<false><<<(n_hits + 255) / 256, 256, 0, st>>>(p->d_best_key, p->d_staged, n_hits, d_hit_to_cand, d_cand_nhits);
    HOUGH_CUDA_TRY(cudaGetLastError());
    hough_count_launches(launches);
    return HOUGH_OK;
}

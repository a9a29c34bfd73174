// walk.cuh -- the column walk shared by the vote (A2/A3, vote.cu) and the hit association (A5, assign.cu).
//
// One CTA owns the tile (event e, d0 slice k, phi0 columns [c0, c0 + cols)) in shared memory:
//   WALK_VOTE   : the tile is that part of the accumulator (two 16-bit bins per word, or 32-bit bins); votes
//                 are shared-memory atomics, the tile is written to HBM exactly once (no global atomic; this
//                 also implements "overwrite", S8).
//   WALK_ASSIGN : the tile holds, per bin, the best candidate of the event within assoc_dj bins of it along
//                 q/pT ("dilated" entries, built from the candidate list in the prologue); every vote position
//                 of a hit needs ONE probe; the best D8 key per (hit, tile) is published with one atomicMax.
//
// Work mapping: lane = hit.  A warp takes 32 consecutive staged hits of one radius class (same window length,
// neighbouring azimuth thanks to the (class, sector) sort of stage.cu); every lane walks the `steps` columns of
// its own window.  Lanes stay converged because `steps` is a property of (class, k).
//
// Bin index per (hit, column): DESIGN.md "Fast path".  The prescribed D3 sequence costs ~30 issue slots
// (IEEE reciprocal, unfused multiplies).  The walk first evaluates the same real-valued function with FMAs and
// MUFU.RCP (t~) together with a bound m on |t~ - t_D3| (first-order rounding analysis of BOTH sequences, x3
// safety); if floor(t~ - m) == floor(t~ + m) the D3 bin is that integer (or certainly out of range) without
// running D3.  Otherwise (about 0.1 % of the evaluations: t within m of a bin edge, NaN/inf, |t| huge) the lane
// runs the exact D3 sequence (d3_exact_bin).  The result is therefore the D3 bin in every case.
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
    int exact_only;                  // 1: never take the fast path (plan option "exact_walk", for bisecting)
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
    b = (b + 15) & ~(size_t)15;
    return b + 128;                                                     // one scratch word per lane (walk_kernel: s_trash)
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

// The exact D3 bin of (hit, column) including the forward test; -1 = no vote.  Out of line: the rare path.
static __device__ __noinline__ int d3_exact_bin(float x, float y, float r2, float cs_c, float cs_s, float d0c, float td0,
                                                float d0sq, float A_f, float qmin, float inv_wq, float nq_f) {
    float w, f;
    d3_wf(x, y, cs_c, cs_s, w, f);
    if (!(f > 0.0f)) return -1;
    return d3_bin_from_w(w, r2, d0c, td0, d0sq, A_f, qmin, inv_wq, nq_f);
}

__device__ __forceinline__ float rcp_approx(float g) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(g));
    return r;
}

__device__ __forceinline__ float rsqrt_approx(float g) {
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(g));
    return r;
}

// atomicAdd on shared memory by shared-window address (no generic-address conversion in the hot loop)
__device__ __forceinline__ void red_shared(unsigned saddr, unsigned val) {
    asm volatile("red.shared.add.u32 [%0], %1;" :: "r"(saddr), "r"(val) : "memory");
}

// Per-tile constants of the fast path (uniform over the CTA).  DESIGN.md "Fast path":
//   t~ - 1/2 = numq * rinv + c0h,   numq = (d0c - w) * inv_wq,   rinv ~ 1 / (A * den),
//   |t~ - t_D3| < m = |rinv| * (elin_h + arel_h * |numq|) + a0,   hm = 1/2 - m.
struct FastK {
    float inv_wq, d0cq, ntd0A, d0sqA, c0h, hm0, e_lin, d0abs, d0sq, A_f;
};

constexpr float WALK_U = 5.9604645e-8f;                 // 2^-24, unit roundoff of fp32
constexpr float WALK_MAGIC = 12582912.0f;               // 1.5 * 2^23: x + MAGIC has rint(x) in its low mantissa bits

__device__ __forceinline__ FastK make_fastk(const HoughConsts& c, float4 d) {
    FastK k;
    k.inv_wq = c.inv_wq;
    k.A_f = c.A_f;
    k.d0cq = d.x * c.inv_wq;
    k.ntd0A = -(d.y * c.A_f);
    k.d0sqA = d.z * c.A_f;
    const float c0 = -(c.qmin * c.inv_wq);
    k.c0h = c0 - 0.5f;
    k.hm0 = 0.5f - 8.0f * WALK_U * (fabsf(c0) + 1.0f);
    k.e_lin = 12.0f * WALK_U * fabsf(c.inv_wq);
    k.d0abs = fabsf(d.x);
    k.d0sq = d.z;
    return k;
}

// Entry of an association tile: (min(votes, VCAP) + 1) << 5 | p,  p = (15 - |dj|) * 2 + (dj < 0), dj = j_cand - j_bin.
// Integer order of entries == D8 order among the candidates of one row that can serve bin j_bin.
template <bool TILE32> struct EntryT {               // 16-bit entries: 11 bits of votes + 1
    static constexpr unsigned VSAT = 2047u;
    typedef unsigned pkey_t;
    static __device__ __forceinline__ pkey_t pkey(unsigned ent, int col) { return ((ent >> 1) << 16) | (unsigned)(0xffff - col); }
    static __device__ __forceinline__ int col_of(pkey_t p) { return 0xffff - (int)(p & 0xffffu); }
    static __device__ __forceinline__ unsigned ent_hi(pkey_t p) { return p >> 16; }
};
template <> struct EntryT<true> {                    // 32-bit entries: 27 bits of votes + 1
    static constexpr unsigned VSAT = (1u << 27) - 1u;
    typedef unsigned long long pkey_t;
    static __device__ __forceinline__ pkey_t pkey(unsigned ent, int col) {
        return ((unsigned long long)(ent >> 1) << 32) | (unsigned)(0x7fffffff - col);
    }
    static __device__ __forceinline__ int col_of(pkey_t p) { return 0x7fffffff - (int)(unsigned)(p & 0xffffffffull); }
    static __device__ __forceinline__ unsigned ent_hi(pkey_t p) { return (unsigned)(p >> 32); }
};

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
    // one scratch word per lane at the end of the block: where the branch-free vote sends the lanes that do not vote
    const unsigned trash_saddr = (unsigned)__cvta_generic_to_shared(
        smem_raw + walk_smem_bytes(slab_cols, stride, nc) - 128 + 4 * lane);
    unsigned short* s_tile16 = reinterpret_cast<unsigned short*>(s_tile);
    const unsigned tile_saddr = (unsigned)__cvta_generic_to_shared(s_tile);

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
        const int steps = w.y & 0x3fffffff;
        s_lo[cl] = lo;
        s_steps[cl] = w.y;                               // bit 30: every column of the window is forward (f > 0)
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
    // association: does any candidate of the tile exceed the entry's vote field?  (then: exact probing, below)
    bool legacy = false;
    if (MODE == WALK_ASSIGN) {
        int sat = 0;
        for (int ci = cand_first + tid; ci < cand_end; ci += WALK_THREADS)
            sat |= ((unsigned)__ldg(&a.cands[ci].votes) + 1u >= EntryT<TILE32>::VSAT) ? 1 : 0;
        legacy = __syncthreads_or(sat) != 0 || a.exact_only != 0;
    } else {
        __syncthreads();
    }
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
    if (MODE == WALK_ASSIGN) {
        if (legacy) {                                   // votes + 1 at the candidates' own bins
            for (int ci = cand_first + tid; ci < cand_end; ci += WALK_THREADS) {
                const int4 q = __ldg(reinterpret_cast<const int4*>(a.cands + ci));          // event, k, i, j
                const unsigned v = (unsigned)__ldg(&a.cands[ci].votes) + 1u;
                const int col = q.z - c0;
                if (TILE32) s_tile[col * stride + q.w] = v;
                else s_tile16[col * stride * 2 + q.w] = (unsigned short)min(v, 65535u);
            }
        } else {                                        // dilated entries: max over the candidates within assoc_dj
            const int dj = a.assoc_dj;
            for (int ci = cand_first + tid; ci < cand_end; ci += WALK_THREADS) {
                const int4 q = __ldg(reinterpret_cast<const int4*>(a.cands + ci));
                const unsigned v = ((unsigned)__ldg(&a.cands[ci].votes) + 1u) << 5;
                const int col = q.z - c0;
                for (int jb = max(q.w - dj, 0); jb <= min(q.w + dj, nq - 1); ++jb) {
                    const int d = q.w - jb;                                                  // j_cand - j_bin
                    const unsigned ent = v | (unsigned)((15 - abs(d)) * 2 + (d < 0 ? 1 : 0));
                    if (TILE32) {
                        atomicMax(s_tile + col * stride + jb, ent);
                    } else {
                        const int h = col * stride * 2 + jb;
                        uint32_t* wp = s_tile + (h >> 1);
                        const int sh = (h & 1) * 16;
                        uint32_t old = *wp;
                        while (((old >> sh) & 0xffffu) < ent) {
                            const uint32_t nw = (old & ~(0xffffu << sh)) | (ent << sh);
                            const uint32_t prev = atomicCAS(wp, old, nw);
                            if (prev == old) break;
                            old = prev;
                        }
                    }
                }
            }
        }
    }
    __syncthreads();

    // ---- main loop: 32-hit batches, static round-robin over the CTA's warps ----
    const int n_batches = s_seg_pref[2 * nc];
    const float4 d = __ldg(c.d0t + k);
    const FastK fk = make_fastk(c, d);
    const bool exact_only = a.exact_only != 0 || nq > (1 << 20);      // the rint trick needs |t| < 2^22
    const unsigned row_lin0 = (unsigned)(k * nphi + c0) * (unsigned)nq;   // linear bin of (k, c0, 0) inside the event
    int seg = 0;                                        // batches ascend per warp: a running segment pointer
    for (int bt = warp; bt < n_batches; bt += WALK_WARPS) {
        while (s_seg_pref[seg + 1] <= bt) ++seg;         // largest segment with seg_pref[seg] <= bt (seg_pref[2nc] = n_batches > bt)
        const int in_seg = (bt - s_seg_pref[seg]) * 32 + lane;
        const bool active = in_seg < s_seg_cnt[seg];
        const int cl = seg >> 1;
        const int steps_w = s_steps[cl];
        const int steps = steps_w & 0x3fffffff;
        const bool fwd_safe = (steps_w >> 30) & 1;
        float4 hv = make_float4(1.f, 0.f, 0.f, 0.f);
        if (active) hv = __ldg(a.staged + ev_begin + s_seg_start[seg] + in_seg);
        const float x = hv.x, y = hv.y;
        const float r2 = d3_r2(x, y);
        // fast-path per-hit terms
        const float r2Ak = __fmaf_rn(r2, fk.A_f, fk.d0sqA);              // g~ = ntd0A * w + r2Ak
        const float L = fabsf(x) + fabsf(y);
        const float elin_h = fk.e_lin * (L + fk.d0abs);
        float arel_h;
        {
            const float S = __fmaf_rn(8.0f * fk.d0abs, L, r2 + fk.d0sq);
            // den >= (r - |d0|)^2; r from the approximate reciprocal square root (2 ulp), shrunk by 2^-20 r
            const float rr = r2 * rsqrt_approx(r2);
            const float dr = fmaxf(fabsf(rr - fk.d0abs) - 9.5367432e-7f * rr, 0.0f);
            arel_h = WALK_U * __fmaf_rn(6.0f, S * rcp_approx(dr * dr), 24.0f);
            if (!(arel_h < 1.0f)) arel_h = 1.0f;                          // r ~ |d0| (or NaN): every evaluation goes exact
        }
        int i_lo = (int)ceilf(hv.z + s_lo[cl]);
        if (i_lo < 0) i_lo += nphi;
        if (i_lo >= nphi) i_lo -= nphi;
        if (!(i_lo >= 0 && i_lo < nphi)) i_lo = 0;
        int col, t_cnt, my_b = 0, my_n;
        if (FULLPHI) {
            col = i_lo;
            t_cnt = steps;
            my_n = 0;
        } else {
            int dd = i_lo - c0;                          // column relative to the tile, cyclic
            if (dd < 0) dd += nphi;
            const bool inside = dd < cols;
            int t_begin = inside ? 0 : nphi - dd;
            int t_end = inside ? min(steps, cols - dd) : min(steps, nphi - dd + cols);
            if (steps + cols > nphi) { t_begin = 0; t_end = steps; }       // a window could re-enter the tile
            if (!active || t_begin >= t_end) { t_begin = 0x3fffffff; t_end = 0; }
            const int tb = __reduce_min_sync(0xffffffffu, t_begin);
            const int te = __reduce_max_sync(0xffffffffu, t_end);
            if (tb >= te) continue;
            col = dd + tb;
            if (col >= nphi) col -= nphi;
            t_cnt = te - tb;
            my_b = t_begin - tb;                         // this lane's own part of the warp's column range
            my_n = t_end > t_begin ? t_end - t_begin : 0;
        }

        unsigned long long best = 0ull;                  // legacy association: full D8 key
        // dilated association: (entry >> 1) above ~column (equal votes and |dj| in two columns: the smaller linear
        // bin wins, D8); the entry's sign bit travels with the q/pT bin in bestj
        typename EntryT<TILE32>::pkey_t bestp = 0;
        int bestj = 0;

// what one vote position (tile column `col`, q/pT bin J >= 0) does
#define WALK_AT(COL, J)                                                                                              \
        do {                                                                                                    \
            if (MODE == WALK_VOTE) {                                                                            \
                if (TILE32) atomicAdd(s_tile + (COL) * stride + (J), 1u);                                         \
                else atomicAdd(s_tile + (COL) * stride + ((J) >> 1), (unsigned)((J) & 1) * 0xffffu + 1u);         \
            } else if (!legacy) {                                                                               \
                const unsigned ent_ = TILE32 ? s_tile[(COL) * stride + (J)] : (unsigned)s_tile16[(COL) * stride * 2 + (J)]; \
                const typename EntryT<TILE32>::pkey_t p_ = EntryT<TILE32>::pkey(ent_, (COL));                    \
                if (p_ > bestp) { bestp = p_; bestj = ((J) << 1) | (int)(ent_ & 1u); }                          \
            } else {                                                                                            \
                const int j0_ = max((J) - a.assoc_dj, 0), j1_ = min((J) + a.assoc_dj, nq - 1);                  \
                for (int jj = j0_; jj <= j1_; ++jj) {                                                           \
                    unsigned v_;                                                                                \
                    if (TILE32) v_ = s_tile[(COL) * stride + jj];                                                 \
                    else v_ = s_tile16[(COL) * stride * 2 + jj];                                                  \
                    if (v_) {                                                                                   \
                        if (!TILE32 && v_ == 65535u) /* saturated 16-bit entry: votes from the record */        \
                            v_ = walk_lookup_votes(a.cands, cand_first, cand_end, c0 + (COL), jj) + 1u;           \
                        const unsigned long long key_ = walk_key(v_ - 1u, abs(jj - (J)), row_lin0 + (unsigned)((COL) * nq + jj)); \
                        best = key_ > best ? key_ : best;                                                       \
                    }                                                                                           \
                }                                                                                               \
            }                                                                                                   \
        } while (0)

// the same under predicate P; the vote is branch-free: lanes with P false add to their scratch word (J arbitrary)
#define WALK_AT_IF(P, COL, J)                                                                                   \
        do {                                                                                                    \
            if (MODE == WALK_VOTE) {                                                                            \
                if (TILE32) red_shared((P) ? tile_saddr + (unsigned)(((COL) * stride + (J)) << 2) : trash_saddr, 1u); \
                else red_shared((P) ? tile_saddr + (unsigned)(((COL) * stride + ((J) >> 1)) << 2) : trash_saddr, \
                                __funnelshift_l(0u, 1u, (unsigned)(J) << 4));                                   \
            } else {                                                                                            \
                if (P) WALK_AT(COL, J);                                                                         \
            }                                                                                                   \
        } while (0)

        if (exact_only || (MODE == WALK_ASSIGN && legacy)) {
            // the D3 sequence at every column of the window (bisecting option / saturated association tiles)
            for (int t = 0; t < t_cnt; ++t) {
                const bool in_tile = FULLPHI ? true : (col < cols);
                const bool mine = FULLPHI ? active : (in_tile && (unsigned)(t - my_b) < (unsigned)my_n);
                if (mine) {
                    const float2 cs = s_cs[col];
                    const int j = d3_exact_bin(x, y, r2, cs.x, cs.y, d.x, d.y, d.z, c.A_f, c.qmin, c.inv_wq, c.nq_f);
                    if (j >= 0) WALK_AT(col, j);
                }
                ++col;
                if (col == nphi) col = 0;
            }
        } else {
            // Fast path.  Lanes whose t~ lies within m of a bin edge (or is NaN) are recorded in `slowmask` and
            // redone with the exact D3 sequence after each chunk of 32 columns, so the hot loop has no branch.
            for (int tb0 = 0; tb0 < t_cnt; tb0 += 32) {
                const int n_it = min(32, t_cnt - tb0);
                const int col_chunk = col;
                // inactive lanes (tail of a batch): range test never passes, bin decision always "sure"
                const unsigned nq_l = active ? (unsigned)nq : 0u;
                const float hm0_l = active ? fk.hm0 : 3.0e38f;
                unsigned slowmask = 0u;                  // bit (n_it - 1 - i): column i of the chunk needs the exact path
                if (fwd_safe) {
#pragma unroll 2
                    for (int t = tb0; t < tb0 + n_it; ++t) {
                        const bool in_tile = FULLPHI ? true : (col < cols);
                        const bool mine = FULLPHI ? true : (in_tile && (unsigned)(t - my_b) < (unsigned)my_n);
                        const float2 cs = s_cs[in_tile ? col : 0];
                        const float w = __fmaf_rn(y, cs.x, -__fmul_rn(x, cs.y));
                        const float numq = __fmaf_rn(-w, fk.inv_wq, fk.d0cq);
                        const float rinv = rcp_approx(__fmaf_rn(fk.ntd0A, w, r2Ak));
                        const float th = __fmaf_rn(numq, rinv, fk.c0h);                        // t~ - 1/2
                        const float hm = __fmaf_rn(__fmaf_rn(arel_h, fabsf(numq), elin_h), -fabsf(rinv), hm0_l);
                        const float yb = __fadd_rn(th, WALK_MAGIC);
                        const float dlt = __fsub_rn(th, __fsub_rn(yb, WALK_MAGIC));             // (t~ - 1/2) - J
                        const int jf = __float_as_int(yb) - __float_as_int(WALK_MAGIC);         // J = rint(t~ - 1/2)
                        const bool sure = fabsf(dlt) < hm;                                      // J <= t_D3 < J + 1
                        WALK_AT_IF(mine && sure && (unsigned)jf < nq_l, col, jf);
                        slowmask = (slowmask << 1) | ((mine && !sure) ? 1u : 0u);
                        ++col;
                        if (col == nphi) col = 0;
                    }
                } else {
#pragma unroll 2
                    for (int t = tb0; t < tb0 + n_it; ++t) {
                        const bool in_tile = FULLPHI ? true : (col < cols);
                        const bool mine = FULLPHI ? true : (in_tile && (unsigned)(t - my_b) < (unsigned)my_n);
                        const float2 cs = s_cs[in_tile ? col : 0];
                        const float w = __fmaf_rn(y, cs.x, -__fmul_rn(x, cs.y));
                        const bool fwd = __fadd_rn(__fmul_rn(x, cs.x), __fmul_rn(y, cs.y)) > 0.0f;   // the exact D3 forward test
                        const float numq = __fmaf_rn(-w, fk.inv_wq, fk.d0cq);
                        const float rinv = rcp_approx(__fmaf_rn(fk.ntd0A, w, r2Ak));
                        const float th = __fmaf_rn(numq, rinv, fk.c0h);
                        const float hm = __fmaf_rn(__fmaf_rn(arel_h, fabsf(numq), elin_h), -fabsf(rinv), hm0_l);
                        const float yb = __fadd_rn(th, WALK_MAGIC);
                        const float dlt = __fsub_rn(th, __fsub_rn(yb, WALK_MAGIC));
                        const int jf = __float_as_int(yb) - __float_as_int(WALK_MAGIC);
                        const bool sure = fabsf(dlt) < hm;
                        WALK_AT_IF(mine && fwd && sure && (unsigned)jf < nq_l, col, jf);
                        slowmask = (slowmask << 1) | ((mine && fwd && !sure) ? 1u : 0u);
                        ++col;
                        if (col == nphi) col = 0;
                    }
                }
                if (!active) slowmask = 0u;
                if (__any_sync(0xffffffffu, slowmask != 0u)) {
                    while (slowmask) {
                        const int bpos = __ffs(slowmask) - 1;
                        slowmask &= slowmask - 1u;
                        int cc = col_chunk + (n_it - 1 - bpos);
                        if (cc >= nphi) cc -= nphi;
                        const float2 cs = s_cs[cc];
                        const int j = d3_exact_bin(x, y, r2, cs.x, cs.y, d.x, d.y, d.z, c.A_f, c.qmin, c.inv_wq, c.nq_f);
                        if (j >= 0) WALK_AT(cc, j);
                    }
                }
            }
        }
#undef WALK_AT_IF
#undef WALK_AT
        if (MODE == WALK_ASSIGN) {
            if (!legacy) {
                const unsigned eh = EntryT<TILE32>::ent_hi(bestp);      // entry >> 1: votes + 1 above (15 - |dj|)
                if (eh) {
                    const int bcol = EntryT<TILE32>::col_of(bestp);
                    const int adj = 15 - (int)(eh & 15u);
                    const int jc = (bestj >> 1) + ((bestj & 1) ? -adj : adj);
                    best = walk_key((eh >> 4) - 1u, adj, row_lin0 + (unsigned)(bcol * nq + jc));
                }
            }
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
    a.exact_only = p->exact_walk;
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

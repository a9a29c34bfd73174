// walk.cuh -- the column walk shared by the vote (A2/A3, vote.cu) and the hit association (A5, assign.cu).
//
// One CTA owns the tile (event e, d0 slice k, phi0 columns [c0, c0 + cols)) in shared memory:
//   WALK_VOTE   : the tile is that part of the accumulator; votes are shared-memory atomics, the tile is written
//                 to HBM exactly once (no global atomic; this also implements "overwrite", S8).
//   WALK_ASSIGN : the tile holds, per bin, the best candidate of the event within assoc_dj bins of it along
//                 q/pT ("dilated" entries, built from the candidate list in the prologue); every vote position
//                 of a hit needs ONE probe; the best D8 key per (hit, tile) is published with one atomicMax.
//
// Tile layout.  A row has nq + 2 slots h = J + 1: the q/pT bins J = 0..nq-1 and one
// GUARD slot at each end (J = -1 and J = nq) that absorbs the fast path's "one bin outside" results, followed by
// WALK_DUMP dump slots for everything further out; guard and dump slots are never flushed.  Packed tiles (16-bit
// bins) store the two columns of an even/odd column PAIR in one 32-bit word per slot (low half = even column, high
// half = odd column), so the increment is the constant 1 or 65536 and the address is pair_row + 4 h.  32-bit tiles
// store one word per (column, slot).
//
// Work mapping: lane = hit.  A warp takes 32 consecutive staged hits of one radius class (same window length,
// neighbouring azimuth thanks to the (class, sector) sort of stage.cu); every lane walks the columns of its own
// window TWO AT A TIME with packed fp32x2 arithmetic (FFMA2 / FADD2 on sm_100a).
//
// Bin index per (hit, column): DESIGN.md "Fast path".  The prescribed D3 sequence costs ~30 issue slots (IEEE
// reciprocal, unfused multiplies).  The walk evaluates the same real-valued function with FMAs and MUFU.RCP (t~)
// and owns, per (radius class, d0 slice), a bound m on |t~ - t_D3| (first-order rounding analysis of BOTH sequences
// with a safety factor); if t~ is further than m from a bin edge the D3 bin is floor(t~) (or certainly out of range)
// without running D3.  The per-column quantity w = y cos - x sin comes from a recurrence in registers (no table read in
// the hot loop, see "Recurrence" below).  The hot loop has no branch: a column pair with an uncertain evaluation
// (about 0.9 % of the pairs) sends both its votes / probes to guard slot 0 of their rows and goes to the warp's small
// shared-memory queue, which the whole warp drains 32 pairs at a time with the exact D3 sequence (d3_exact_bin) for both
// columns.  Classes whose bound is useless (r ~ |d0|, the open-ended
// last class where non-finite coordinates land), classes whose window is not certainly forward, and the plan option
// "exact_walk" take the exact sequence at every column.  The result is therefore the D3 bin in every case.
#pragma once

#include <cstdlib>
#include <type_traits>

#include "common.cuh"

constexpr int WALK_VOTE = 0;
constexpr int WALK_ASSIGN = 1;
// threads per CTA: the vote walk runs best with 10 warps at 64 registers, the association walk (more live state) with
// 8 warps at 80 registers (profiles/r1_final.md)
__host__ __device__ constexpr int walk_threads(int mode) { return mode == 0 ? 320 : 256; }
constexpr int WALK_MAX_WARPS = 10;
constexpr int WALK_CHUNK_PAIRS = 32;             // column pairs per chunk = the bits of the redo mask
constexpr int WALK_WQ_CAP = 64;                  // entries of a warp's redo queue: < 32 waiting + up to 32 new ones per round

struct WalkArgs {
    const float4* staged;            // [n_hits] staged hits (stage.cu)
    const int32_t* off;              // [n_events + 1] event offsets
    const int32_t* key_start;        // [n_events][n_keys + 1] exclusive key starts
    int n_slabs, slab_cols, stride;  // tile shape (slab_cols even; stride = words per row / pair row, odd)
    int exact_only;                  // 1: never take the fast path (plan option "exact_walk", for bisecting)
    float m_scale;                   // 1; the self-check build's HOUGH_DEBUG_M_SCALE scales the bound m (margin probe, profiles/r2_walk.md)
    // WALK_VOTE
    void* accum;
    // WALK_ASSIGN
    const hough_candidate* cands;
    const int2* slice;               // [n_events * n_d0 * n_slabs] {first, end} candidate of each tile
    int assoc_dj;
    unsigned long long* best_key;    // [n_hits] by original hit index
    const uint8_t* keep;             // optional [capacity]: only candidates with keep != 0 take part (D12 re-assignment round)
};

constexpr int WALK_DUMP = 4;                     // dump slots per row: where results outside [-1, nq] are added (by lane & 3)
__host__ __device__ inline int walk_row_stride(int nq) { return (nq + 2 + WALK_DUMP) | 1; }

__host__ __device__ inline size_t walk_tile_words(int cols, int stride, bool tile32) {
    return tile32 ? (size_t)cols * stride : (size_t)((cols + 1) / 2) * stride;
}

__host__ __device__ inline size_t walk_smem_bytes(int cols, int stride, bool tile32, int n_class, bool fullphi) {
    size_t b = (walk_tile_words(cols, stride, tile32) * 4 + 15) & ~(size_t)15;
    b += (size_t)n_class * 16;                                          // per class: window, error bound
    b += ((size_t)n_class * (fullphi ? 1 : 2) + 1) * 16;                // segments (a full-phi tile has one per class)
    b += (size_t)WALK_MAX_WARPS * WALK_WQ_CAP * 4;                      // redo queues
    return b + 128;                                                     // one scratch word per lane (walk_kernel: trash_saddr)
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
                                                float d0sq, float A_f, float qmin, float inv_wq, float nq_f, bool line) {
    float w, f;
    d3_wf(x, y, cs_c, cs_s, w, f);
    if (!(f > 0.0f)) return -1;
    return d3_bin_from_w(w, r2, d0c, td0, d0sq, A_f, qmin, inv_wq, nq_f, line);
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

// ---- packed fp32x2 arithmetic (sm_100a: FFMA2 / FADD2, two fp32 lanes per issue slot) ----
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk2(f32x2 v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
    f32x2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) {
    f32x2 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}

// shared-memory accesses by shared-window address (no generic-address conversion in the hot loop)
__device__ __forceinline__ void red_shared(unsigned saddr, unsigned val) {
    asm volatile("red.shared.add.u32 [%0], %1;" :: "r"(saddr), "r"(val) : "memory");
}
__device__ __forceinline__ unsigned lds_u16(unsigned saddr) {
    unsigned short v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(saddr));
    return (unsigned)v;
}
__device__ __forceinline__ unsigned lds_u32(unsigned saddr) {
    unsigned v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(saddr));
    return v;
}
// base + 4 * idx as one IMAD (keeps the compiler from re-associating the address into three instructions)
__device__ __forceinline__ unsigned addr_w(unsigned base, unsigned idx) {
    unsigned r;
    asm("mad.lo.u32 %0, %1, 4, %2;" : "=r"(r) : "r"(idx), "r"(base));
    return r;
}

constexpr float WALK_U = 5.9604645e-8f;                 // 2^-24, unit roundoff of fp32
constexpr float WALK_MAGIC = 12582912.0f;               // 1.5 * 2^23: x + MAGIC has rint(x) in its low mantissa bits
constexpr int WALK_MAGIC_BITS = 0x4B400000;

// Per-tile constants of the fast path (uniform over the CTA).  DESIGN.md "Fast path":
//   t~ - 1/2 = numq * rinv + c0h,   numq = ny c + nx s + d0cq = (d0c - w) inv_wq,   rinv ~ 1 / (gy c + gx s + r2Ak) = 1 / (A den)
//   |t~ - t_D3| < m_h = rmax_h * elin_h + arel_h * Tmax + a0   for every column whose t~ lies in [-1, nq + 1]
struct FastK {
    float inv_wq, d0cq, ntd0A, d0sqA, c0h, a0, e_lin, d0abs, d0sq, A_f, inv_A_abs, t_max;
    float nq_s;       // numq = nq_s (y c - x s) + d0cq:  -inv_wq (helix: (d0c - w) inv_wq),  +inv_wq (line: w inv_w)
    bool usable;
    bool line;        // HOUGH_MODEL_LINE: t~ = w inv_w + c0 -- the same loop with A den == 1 (ntd0A = A = 0, d0sqA = 1)
};

__device__ __forceinline__ FastK make_fastk(const HoughConsts& c, float4 d) {
    FastK k;
    k.inv_wq = c.inv_wq;
    k.A_f = c.A_f;
    k.d0cq = d.x * c.inv_wq;
    k.ntd0A = -(d.y * c.A_f);
    k.d0sqA = d.z * c.A_f;
    const float c0 = -(c.qmin * c.inv_wq);
    k.c0h = c0 - 0.5f;
    k.a0 = 8.0f * WALK_U * (fabsf(c0) + 1.0f);
    k.e_lin = 12.0f * WALK_U * fabsf(c.inv_wq);
    k.d0abs = fabsf(d.x);
    k.d0sq = d.z;
    k.inv_A_abs = 1.0f / fabsf(c.A_f);
    k.t_max = fmaxf(fabsf(c0), fabsf(c.nq_f - c0)) + 2.0f;
    // the rint trick needs |t| < 2^22; a zero / non-finite field constant or range has no usable bound
    k.line = c.model != 0;
    k.nq_s = k.line ? c.inv_wq : -c.inv_wq;
    if (k.line) { k.inv_A_abs = 1.0f; k.ntd0A = 0.0f; k.A_f = 0.0f; k.d0sqA = 1.0f; }   // no denominator: A den == 1
    k.usable = c.n_qpt < (1 << 20) && k.inv_A_abs < 3.0e38f && k.t_max < 4.0e6f && k.e_lin < 3.0e38f;
    return k;
}

// ---- Recurrence.  Both A den and the numerator are affine in ONE per-column quantity,
//   w_i = y cos_i - x sin_i = r sin(phi_hit - theta_i):     A den ~ ntd0A w + r2Ak,    numq ~ nq_s w + d0cq,
// and along the columns of a pair walk (step 2 columns = angle 2 wphi) w obeys  w_{n+1} = 2 cos(2 wphi) w_n - w_{n-1}.
// In Reinsch's difference form (stable for small angles):  d_{n+1} = d_n - kappa w_n,  w_{n+1} = w_n + d_{n+1},
// kappa = 4 sin^2(wphi): one FFMA2 + one FADD2 per column pair and NO table read in the hot loop.  The walk
// re-initialises (w, d) from the cos/sin table at the first pair of every chunk of WALK_CHUNK_PAIRS pairs:
//   w_0 = y c - x s at the pair's two columns,   d_0 = w_0 - w_{-1} = -2 sin(wphi) (x c' + y s') with (c', s') of the column
//   before each (the half-way column of the step) -- no cancellation.
// The rounding error the recurrence accumulates over a chunk enters the bound m through Ew (walk_kernel prologue).
// Nothing is ever replayed: a pair the fast path cannot decide votes into guard slot 0 and is redone with the exact D3
// sequence from the table (walk_kernel "redo"), so the recurrence only has to stay inside the bound, not be reproducible.
struct WRec { f32x2 w2, d2; };
__device__ __forceinline__ WRec wrec_init(const HoughConsts& c, float x, float y, int ca) {      // ca: absolute column, even
    HOUGH_CHECK(ca >= 0 && ca + 1 < c.n_phi && (ca & 1) == 0);
    const float4 T = __ldg(reinterpret_cast<const float4*>(c.cs + ca));                          // {cosA, sinA, cosB, sinB}
    const float2 M = __ldg(c.cs + ca - 1);                                                        // the column before A (cs[-1] = cs[n_phi - 1])
    const float wA = __fmaf_rn(y, T.x, -__fmul_rn(x, T.y));
    const float wB = __fmaf_rn(y, T.z, -__fmul_rn(x, T.w));
    const float fM = __fmaf_rn(y, M.y, __fmul_rn(x, M.x));
    const float fA = __fmaf_rn(y, T.y, __fmul_rn(x, T.x));
    WRec r;
    r.w2 = pk2(wA, wB);
    r.d2 = pk2(-__fmul_rn(c.sd2, fM), -__fmul_rn(c.sd2, fA));
    return r;
}
__device__ __forceinline__ void wrec_step(WRec& r, f32x2 nkap2) {
    r.d2 = fma2(nkap2, r.w2, r.d2);
    r.w2 = add2(r.w2, r.d2);
}
// The fast-path bin of ONE column from the cos/sin table (no recurrence): true and J = the D3 bin when t~ is further than
// the class's bound from a bin edge (the bound covers this sequence as well: its w carries 2 roundings, Ew allows for more).
__device__ __forceinline__ bool fast_bin_direct(const FastK& fk, float x, float y, float r2Ak, float2 cs, float hm, int& J) {
    const float w = __fmaf_rn(y, cs.x, -__fmul_rn(x, cs.y));
    const float g = __fmaf_rn(fk.ntd0A, w, r2Ak);
    const float n = __fmaf_rn(fk.nq_s, w, fk.d0cq);
    const float th = __fmaf_rn(n, rcp_approx(g), fk.c0h);
    const float yb = __fadd_rn(th, WALK_MAGIC);
    const float dl = __fsub_rn(th, __fadd_rn(yb, -WALK_MAGIC));
    J = __float_as_int(yb) - WALK_MAGIC_BITS;
    return fabsf(dl) < hm;
}
// t~ - 1/2 of the pair's two columns
__device__ __forceinline__ f32x2 wrec_th(f32x2 w2, f32x2 ntd0A2, f32x2 r2Ak2, f32x2 nqs2, f32x2 d0cq2, f32x2 c0h2) {
    const f32x2 g2 = fma2(ntd0A2, w2, r2Ak2);
    const f32x2 n2 = fma2(nqs2, w2, d0cq2);
    float gA, gB;
    upk2(g2, gA, gB);
    return fma2(n2, pk2(rcp_approx(gA), rcp_approx(gB)), c0h2);
}
// Entry of an association tile: (min(votes, VCAP) + 1) << 5 | p,  p = (15 - |dj|) * 2 + (dj < 0), dj = j_cand - j_bin.
// Integer order of entries == D8 order among the candidates of one row that can serve bin j_bin.
template <bool TILE32> struct EntryT {               // 16-bit entries: 11 bits of votes + 1
    static constexpr unsigned VSAT = 2047u;
    typedef unsigned pkey_t;
    static constexpr unsigned CINV0 = 0xffffu;
    static __device__ __forceinline__ pkey_t pkey(unsigned ent, int col) { return ((ent >> 1) << 16) | (unsigned)(0xffff - col); }
    static __device__ __forceinline__ pkey_t pkey_inv(unsigned ent, unsigned cinv) { return ((ent << 15) & 0xffff0000u) | cinv; }
    static __device__ __forceinline__ int col_of(pkey_t p) { return 0xffff - (int)(p & 0xffffu); }
    static __device__ __forceinline__ unsigned ent_hi(pkey_t p) { return p >> 16; }
};
template <> struct EntryT<true> {                    // 32-bit entries: 27 bits of votes + 1
    static constexpr unsigned VSAT = (1u << 27) - 1u;
    typedef unsigned long long pkey_t;
    static constexpr unsigned CINV0 = 0x7fffffffu;
    static __device__ __forceinline__ pkey_t pkey(unsigned ent, int col) {
        return ((unsigned long long)(ent >> 1) << 32) | (unsigned)(0x7fffffff - col);
    }
    static __device__ __forceinline__ pkey_t pkey_inv(unsigned ent, unsigned cinv) {
        return ((unsigned long long)(ent >> 1) << 32) | cinv;
    }
    static __device__ __forceinline__ int col_of(pkey_t p) { return 0x7fffffff - (int)(unsigned)(p & 0xffffffffull); }
    static __device__ __forceinline__ unsigned ent_hi(pkey_t p) { return (unsigned)(p >> 32); }
};

// ---- tile accessors by (tile column, q/pT bin J in [0, nq)) ----
template <bool TILE32>
__device__ __forceinline__ void tile_vote(uint32_t* s_tile, int stride, int col, int J) {
    HOUGH_CHECK(col >= 0 && J >= 0 && J + 1 < stride);
    if (TILE32) atomicAdd(s_tile + col * stride + J + 1, 1u);
    else atomicAdd(s_tile + (col >> 1) * stride + J + 1, 1u << (16 * (col & 1)));
}
// +1 / -1 at slot `slot` (guard slots included) of tile column col
template <bool TILE32>
__device__ __forceinline__ void tile_add_slot(uint32_t* s_tile, int stride, int col, unsigned slot, int delta) {
    if (TILE32) atomicAdd(s_tile + col * stride + slot, (unsigned)delta);
    else atomicAdd(s_tile + (col >> 1) * stride + slot, (unsigned)delta << (16 * (col & 1)));
}
template <bool TILE32>
__device__ __forceinline__ unsigned tile_entry(const uint32_t* s_tile, int stride, int col, int J) {
    HOUGH_CHECK(col >= 0 && J >= 0 && J + 1 < stride);
    if (TILE32) return s_tile[col * stride + J + 1];
    return (unsigned)reinterpret_cast<const unsigned short*>(s_tile)[(((col >> 1) * stride + J + 1) << 1) + (col & 1)];
}

// What one exact vote position (tile column col, q/pT bin J in [0, nq)) does.  Association: the D8 key of the best
// candidate serving the position is folded into `best`.
template <int MODE, bool TILE32>
__device__ __forceinline__ void walk_apply(uint32_t* s_tile, int stride, int nq, int col, int J, bool legacy, int assoc_dj,
                                           const hough_candidate* __restrict__ cands, int cand_first, int cand_end, int c0,
                                           unsigned row_lin0, unsigned long long& best) {
    if (MODE == WALK_VOTE) {
        tile_vote<TILE32>(s_tile, stride, col, J);
    } else if (!legacy) {
        const unsigned ent = tile_entry<TILE32>(s_tile, stride, col, J);
        if (ent) {
            const int adj = 15 - (int)((ent >> 1) & 15u);
            const int jc = J + ((ent & 1u) ? -adj : adj);
            const unsigned long long key = walk_key((ent >> 5) - 1u, adj, row_lin0 + (unsigned)(col * nq + jc));
            best = key > best ? key : best;
        }
    } else {
        const int j0 = max(J - assoc_dj, 0), j1 = min(J + assoc_dj, nq - 1);
        for (int jj = j0; jj <= j1; ++jj) {
            unsigned v = tile_entry<TILE32>(s_tile, stride, col, jj);
            if (v) {
                if (!TILE32 && v == 65535u)                       // saturated 16-bit entry: votes from the record
                    v = walk_lookup_votes(cands, cand_first, cand_end, c0 + col, jj) + 1u;
                const unsigned long long key = walk_key(v - 1u, abs(jj - J), row_lin0 + (unsigned)(col * nq + jj));
                best = key > best ? key : best;
            }
        }
    }
}

// What the out-of-line rare paths need of the tile (written once per CTA into shared memory).
struct WalkTile {
    uint32_t* s_tile;
    int stride, c0, cand_first, cand_end;
    unsigned row_lin0;
    bool legacy;
};

// Redo of one flagged column pair with the exact D3 sequence.  `sidx` = staged hit, `cc` = tile column of the pair,
// `live` = which columns of the pair belong to the lane's part of the tile.  The hot loop did nothing for a flagged
// pair (no vote, no probe): both columns are decided here.
template <int MODE, bool TILE32>
__device__ __noinline__ void walk_redo_pair(const HoughConsts& c, float4 d, const WalkArgs& a, const WalkTile& tl,
                                            int sidx, int cc, unsigned live) {
    const float4 hv = __ldg(a.staged + sidx);
    const float r2 = d3_r2(hv.x, hv.y);
    int ca = tl.c0 + cc;                                // absolute column of the pair (even)
    if (ca >= c.n_phi) ca -= c.n_phi;
    HOUGH_CHECK(ca >= 0 && ca + 1 < c.n_phi && (ca & 1) == 0 && cc >= 0);
    const float4 T = __ldg(reinterpret_cast<const float4*>(c.cs + ca));     // {cosA, sinA, cosB, sinB}
    unsigned long long best = 0ull;
#pragma unroll
    for (int w = 0; w < 2; ++w) {
        if (!((live >> w) & 1u)) continue;
        const int j = d3_exact_bin(hv.x, hv.y, r2, w ? T.z : T.x, w ? T.w : T.y, d.x, d.y, d.z, c.A_f, c.qmin, c.inv_wq, c.nq_f,
                                   c.model != 0);
        if (j >= 0)
            walk_apply<MODE, TILE32>(tl.s_tile, tl.stride, c.n_qpt, cc + w, j, tl.legacy, a.assoc_dj, a.cands, tl.cand_first,
                                     tl.cand_end, tl.c0, tl.row_lin0, best);
    }
    if (MODE == WALK_ASSIGN && best) atomicMax(a.best_key + __float_as_int(hv.w), best);
}

// The exact D3 sequence at every column of one hit's window (classes without a usable fast-path bound, the plan option
// "exact_walk", saturated association tiles).  Out of line: keeps the hot loop's register budget.
template <int MODE, bool TILE32>
__device__ __noinline__ void walk_exact_window(const HoughConsts& c, float4 d, const WalkArgs& a, const WalkTile& tl, int sidx,
                                               int i_lo, int steps, int cols) {
    const float4 hv = __ldg(a.staged + sidx);
    const float r2 = d3_r2(hv.x, hv.y);
    const int nphi = c.n_phi;
    unsigned long long best = 0ull;
    int col = i_lo - tl.c0;                              // column relative to the tile, cyclic
    if (col < 0) col += nphi;
    for (int t = 0; t < steps; ++t) {
        if (col < cols) {
            const float2 T = __ldg(c.cs + tl.c0 + col);
            const int j = d3_exact_bin(hv.x, hv.y, r2, T.x, T.y, d.x, d.y, d.z, c.A_f, c.qmin,
                                       c.inv_wq, c.nq_f, c.model != 0);
            if (j >= 0)
                walk_apply<MODE, TILE32>(tl.s_tile, tl.stride, c.n_qpt, col, j, tl.legacy, a.assoc_dj, a.cands, tl.cand_first,
                                         tl.cand_end, tl.c0, tl.row_lin0, best);
        }
        ++col;
        if (col == nphi) col = 0;
    }
    if (MODE == WALK_ASSIGN && best) atomicMax(a.best_key + __float_as_int(hv.w), best);
}

// Redo queue entry (32 bits): staged index inside the event (18 bits) | pair index inside the tile (10) | live (2)
__device__ __forceinline__ unsigned wq_pack(int in_event, int cc, unsigned live) {
    return (unsigned)in_event | ((unsigned)(cc >> 1) << 18) | (live << 28);
}

// the whole warp redoes n <= 32 queued pairs, one per lane
template <int MODE, bool TILE32>
__device__ __forceinline__ void walk_drain(const HoughConsts& c, float4 d, const WalkArgs& a, const WalkTile& tl,
                                           const unsigned* wq, int n, int ev_begin, int lane) {
    __syncwarp();
    if (lane < n) {
        const unsigned en = wq[lane];
        walk_redo_pair<MODE, TILE32>(c, d, a, tl, ev_begin + (int)(en & 0x3ffffu), (int)((en >> 18) & 0x3ffu) * 2, (en >> 28) & 3u);
    }
    __syncwarp();
}

template <int MODE, bool TILE32, bool OUT16, bool FULLPHI>
__global__ void __launch_bounds__(walk_threads(MODE), 3) walk_kernel(const __grid_constant__ HoughConsts c, const __grid_constant__ WalkArgs a) {
    constexpr int WALK_THREADS = walk_threads(MODE), WALK_WARPS = WALK_THREADS / 32;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ WalkTile s_tl;
    __shared__ int s_meta[2];                           // number of batches of the tile
    // warp-uniform loop state kept in shared memory on purpose ({next batch, segment pointer, queue fill} per warp): at
    // the kernels' register budgets the compiler otherwise spills exactly these to local memory, whose reloads miss the
    // small L1 left beside 3 x 75 KB of tiles (measured: 10 % of the association walk's stall samples)
    __shared__ int s_ws[WALK_MAX_WARPS][4];
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

    uint32_t* s_tile; unsigned* s_wq; float4* s_cls; int4* s_seg;
    {
        unsigned char* q = smem_raw;
        s_tile = reinterpret_cast<uint32_t*>(q);  q += (walk_tile_words(slab_cols, stride, TILE32) * 4 + 15) & ~(size_t)15;
        s_cls = reinterpret_cast<float4*>(q);     q += (size_t)nc * 16;              // {lo_off, bits(steps | flags), hm, -}
        s_seg = reinterpret_cast<int4*>(q);       q += ((size_t)nc * (FULLPHI ? 1 : 2) + 1) * 16;   // {first staged hit, hits, class, first batch}
        s_wq = reinterpret_cast<unsigned*>(q);                                        // [WALK_WARPS][WALK_WQ_CAP]
    }
    unsigned short* s_tile16 = reinterpret_cast<unsigned short*>(s_tile);
    const unsigned tile_saddr = (unsigned)__cvta_generic_to_shared(s_tile);
    const unsigned stride4 = (unsigned)stride * 4u;
    // one scratch word per lane at the end of the block: where slab tiles send the lanes that are past their part
    unsigned char* trash_ptr = smem_raw + walk_smem_bytes(slab_cols, stride, TILE32, nc, FULLPHI) - 128;
    const unsigned trash_saddr = (unsigned)__cvta_generic_to_shared(trash_ptr + 4 * lane);

    int cand_first = 0, cand_end = 0;
    if (MODE == WALK_ASSIGN) {
        const int2 sl = __ldg(a.slice + blockIdx.x);
        cand_first = sl.x; cand_end = sl.y;
        if (cand_first >= cand_end) return;              // no candidate in this tile: nothing to associate
    }
    const float4 d = __ldg(c.d0t + k);
    const FastK fk = make_fastk(c, d);
    const int ev_begin = __ldg(a.off + e);
    const int ev_hits = __ldg(a.off + e + 1) - ev_begin;
    const int32_t* ks = a.key_start + (size_t)e * (c.n_keys + 1);

    // ---- prologue: zero the tile, load tables, list the segments of staged hits that can reach the tile ----
    // association: does any candidate of the tile exceed the entry's vote field?  (then: exact probing, below)
    bool legacy = false;
    if (MODE == WALK_ASSIGN) {
        int sat = 0;
        int any = 0;
        for (int ci = cand_first + tid; ci < cand_end; ci += WALK_THREADS) {
            if (a.keep && !__ldg(a.keep + ci)) continue;
            any = 1;
            sat |= ((unsigned)__ldg(&a.cands[ci].votes) + 1u >= EntryT<TILE32>::VSAT) ? 1 : 0;
        }
        if (a.keep && !__syncthreads_or(any)) return;      // no surviving candidate in this tile
        legacy = __syncthreads_or(sat) != 0 || a.exact_only != 0;
    }
    const bool exact_mode = a.exact_only != 0 || !fk.usable || (MODE == WALK_ASSIGN && legacy);
    {
        uint4* t4 = reinterpret_cast<uint4*>(s_tile);
        const int n4 = (int)((walk_tile_words(cols, stride, TILE32) + 3) >> 2);
        for (int x = tid; x < n4; x += WALK_THREADS) t4[x] = make_uint4(0u, 0u, 0u, 0u);
        if (tid < 32) reinterpret_cast<uint32_t*>(trash_ptr)[tid] = 0u;   // read (as empty entries) by association probes
        if (tid == 0) {
            s_tl.s_tile = s_tile; s_tl.stride = stride; s_tl.c0 = c0; s_tl.cand_first = cand_first;
            s_tl.cand_end = cand_end; s_tl.row_lin0 = (unsigned)(k * nphi + c0) * (unsigned)nq; s_tl.legacy = legacy;
        }
    }
    // per class: column window and the fast path's error bound over the class's radius interval (DESIGN.md "Fast
    // path"): hm = 1/2 - m, or 0 when the class takes the exact sequence at every column
    for (int cl = tid; cl < nc; cl += WALK_THREADS) {
        const int2 w = __ldg(c.win + (size_t)cl * c.n_d0 + k);
        const int steps = w.y & 0x3fffffff;
        const bool fwd_safe = (w.y >> 30) & 1;           // every column of the window (+-2) is forward (f > 0)
        float hm = 0.0f;
        if (!exact_mode && fwd_safe && steps > 0 && cl > 0 && cl + 1 < nc && (FULLPHI || steps + cols + 2 <= nphi)) {
            const float ra = sqrtf(__ldg(c.edge2 + cl)) * 0.999998f, rb = sqrtf(__ldg(c.edge2 + cl + 1)) * 1.000002f;
            const float L = 1.4142137f * rb;                                  // |x| + |y| <= sqrt(2) r
            float dr = (fk.d0abs >= ra && fk.d0abs <= rb) ? 0.0f : fminf(fabsf(ra - fk.d0abs), fabsf(rb - fk.d0abs));
            dr = fmaxf(dr - 1.0e-6f * rb, 0.0f);                              // den >= (r - |d0|)^2 >= dr^2
            const float S = 8.0f * fk.d0abs * L + rb * rb + fk.d0sq;
            const float inv_dr2 = fk.line ? 1.0f : 1.000001f / (dr * dr);       // line model: no denominator at all
            // rounding error of the w recurrence at the end of a chunk (first order, x 1.5): initial values, one rounding of
            // w and of d per pair, d's errors integrated over the remaining pairs
            const float lo_f = __int_as_float(w.x);
            const float Nf = (float)min(WALK_CHUNK_PAIRS, (steps + 3) >> 1);
            const float Th = 2.0f * c.wphi;
            const float wmax = rb * fminf(1.0f, (fmaxf(fabsf(lo_f), fabsf(lo_f + (float)steps)) + 3.0f) * c.wphi);
            const float Ew = 1.5f * WALK_U * (2.0f * L + 4.0f * Nf * Th * L + Nf * wmax + 0.5f * Nf * Nf * Th * rb * (1.0f + Th));
            const float arel = WALK_U * ((fk.line ? 0.0f : 6.0f * S * inv_dr2) + 24.0f) + (fk.line ? 0.0f : 3.0f * fk.d0abs * Ew * inv_dr2);
            const float elin = fk.e_lin * (L + fk.d0abs) + fabsf(fk.inv_wq) * Ew;
            const float m = fk.inv_A_abs * inv_dr2 * elin + arel * fk.t_max + fk.a0;
            if (m < 0.45f) hm = 0.5f - m * a.m_scale;                         // false for NaN / inf
        }
        s_cls[cl] = make_float4(__int_as_float(w.x), __int_as_float(steps), hm, 0.0f);
    }
    // segments (class, sector run) of staged hits whose window can meet the tile: non-empty ones, compacted, with
    // the exclusive prefix of their 32-hit batch counts
    if (warp == 0) {
        int n_out = 0, run = 0;
        const unsigned lt = (1u << lane) - 1u;
        for (int cl0 = 0; cl0 < nc; cl0 += 32) {
            const int cl = cl0 + lane;
            int a0 = 0, n0 = 0, a1 = 0, n1 = 0;
            if (cl < nc) {
                const int2 w = __ldg(c.win + (size_t)cl * c.n_d0 + k);
                const float lo = __int_as_float(w.x);
                const int steps = w.y & 0x3fffffff;
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
            }
            const int b0 = (n0 + 31) >> 5, b1 = (n1 + 31) >> 5;
            const unsigned m0 = __ballot_sync(0xffffffffu, n0 > 0), m1 = __ballot_sync(0xffffffffu, n1 > 0);
            int incl = b0 + b1;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += y;
            }
            const int excl = run + incl - (b0 + b1);
            const int o0 = n_out + __popc(m0 & lt) + __popc(m1 & lt);
            if (n0 > 0) s_seg[o0] = make_int4(a0, n0, cl, excl);
            if (n1 > 0) s_seg[o0 + (n0 > 0 ? 1 : 0)] = make_int4(a1, n1, cl, excl + b0);
            n_out += __popc(m0) + __popc(m1);
            run += __shfl_sync(0xffffffffu, incl, 31);
        }
        if (lane == 0) {
            s_seg[n_out] = make_int4(0, 0, 0, run);      // sentinel: first batch past the end
            s_meta[0] = run;
        }
    }
    if (MODE == WALK_ASSIGN) {
        __syncthreads();                                // the tile is zero
        if (legacy) {                                   // votes + 1 at the candidates' own bins
            for (int ci = cand_first + tid; ci < cand_end; ci += WALK_THREADS) {
                if (a.keep && !__ldg(a.keep + ci)) continue;
                const int4 q = __ldg(reinterpret_cast<const int4*>(a.cands + ci));          // event, k, i, j
                const unsigned v = (unsigned)__ldg(&a.cands[ci].votes) + 1u;
                const int col = q.z - c0;
                if (TILE32) s_tile[col * stride + q.w + 1] = v;
                else s_tile16[(((col >> 1) * stride + q.w + 1) << 1) + (col & 1)] = (unsigned short)min(v, 65535u);
            }
        } else {                                        // dilated entries: max over the candidates within assoc_dj
            const int dj = a.assoc_dj;
            for (int ci = cand_first + tid; ci < cand_end; ci += WALK_THREADS) {
                if (a.keep && !__ldg(a.keep + ci)) continue;
                const int4 q = __ldg(reinterpret_cast<const int4*>(a.cands + ci));
                const unsigned v = ((unsigned)__ldg(&a.cands[ci].votes) + 1u) << 5;
                const int col = q.z - c0;
                for (int jb = max(q.w - dj, 0); jb <= min(q.w + dj, nq - 1); ++jb) {
                    const int dd = q.w - jb;                                                 // j_cand - j_bin
                    const unsigned ent = v | (unsigned)((15 - abs(dd)) * 2 + (dd < 0 ? 1 : 0));
                    if (TILE32) {
                        atomicMax(s_tile + col * stride + jb + 1, ent);
                    } else {
                        uint32_t* wp = s_tile + (col >> 1) * stride + jb + 1;
                        const int sh = (col & 1) * 16;
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
    const int n_batches = s_meta[0];
    const unsigned row_lin0 = (unsigned)(k * nphi + c0) * (unsigned)nq;   // linear bin of (k, c0, 0) inside the event
    const unsigned tile_bytes = (unsigned)(walk_tile_words(cols, stride, TILE32) * 4);   // FULLPHI: the wrap distance
    const unsigned tile_end = tile_saddr + tile_bytes;
    const unsigned tile_alloc_end = tile_saddr + (unsigned)(walk_tile_words(slab_cols, stride, TILE32) * 4);   // (HOUGH_CHECK only)
    (void)tile_alloc_end;
    const f32x2 d0cq2 = pk2(fk.d0cq, fk.d0cq), c0h2 = pk2(fk.c0h, fk.c0h);
    const f32x2 ntd0A2 = pk2(fk.ntd0A, fk.ntd0A), nqs2 = pk2(fk.nq_s, fk.nq_s), nkap2 = pk2(-c.kappa, -c.kappa);
    const f32x2 magic2 = pk2(WALK_MAGIC, WALK_MAGIC), nmagic2 = pk2(-WALK_MAGIC, -WALK_MAGIC);
    const WalkTile& tl = s_tl;                          // what the out-of-line rare paths need of the tile (written in the prologue)
    unsigned* wq = s_wq + warp * WALK_WQ_CAP;           // the warp's redo queue
    volatile int* ws = s_ws[warp];                      // [0] next batch, [1] segment pointer, [2] queue fill (all warp-uniform)
    if (lane == 0) { ws[0] = warp; ws[1] = 0; ws[2] = 0; }
    __syncwarp();
    constexpr bool WS_SMEM = MODE == WALK_ASSIGN;       // the vote walk (64 registers, no spill) keeps them in registers: faster there
    int bt_r = warp, seg_r = 0, wqn_r = 0;
    const unsigned lt = (1u << lane) - 1u;
    const bool wq_ok = ev_hits < (1 << 18) && slab_cols <= 2048;          // entries fit 32 bits (else: redo on the spot)
    const unsigned dump = (unsigned)(lane & (WALK_DUMP - 1));
    for (;;) {
        const int bt = WS_SMEM ? ws[0] : bt_r;
        if (bt >= n_batches) break;
        int seg = WS_SMEM ? ws[1] : seg_r;
        while (s_seg[seg + 1].w <= bt) ++seg;            // last segment with first batch <= bt (the sentinel ends the search)
        if (WS_SMEM) {
            __syncwarp();
            if (lane == 0) { ws[0] = bt + WALK_WARPS; ws[1] = seg; }
        } else {
            bt_r = bt + WALK_WARPS; seg_r = seg;
        }
        HOUGH_CHECK(seg >= 0 && seg < nc * (FULLPHI ? 1 : 2));
        const int4 sg = s_seg[seg];                      // {first staged hit, hits, class, first batch}
        HOUGH_CHECK(sg.z >= 0 && sg.z < nc && sg.x >= 0 && sg.x + sg.y <= ev_hits);
        // A batch = 32 consecutive staged hits of the segment (neighbours in azimuth: their cos/sin pairs sit in adjacent
        // shared-memory words).  Dealing the hits of a segment to the lanes 4 or ~1 tile rows apart was measured and is
        // slower (profiles/r2_walk.md: bank conflicts of the regular spacing outweigh the same-word votes it removes).
        const int in_seg = (bt - sg.w) * 32 + lane;
        const bool active = in_seg < sg.y;
        const float4 cw = s_cls[sg.z];
        const int steps = __float_as_int(cw.y);
        const float hm_c = cw.z;
        const int sidx = ev_begin + sg.x + in_seg;       // index of the lane's staged hit
        float4 hv = make_float4(1.f, 0.f, 0.f, 0.f);
        if (active) hv = __ldg(a.staged + sidx);
        // the warp's next batch is WALK_WARPS batches on: bring its staged hits into L1 while this one is walked (the
        // address only has to be right most of the time; it stays inside the event's staged range)
        {
            const int nxt = sidx + 32 * WALK_WARPS;
            if (nxt < ev_begin + ev_hits) asm volatile("prefetch.global.L1 [%0];" :: "l"(a.staged + nxt));
        }
        const float x = hv.x, y = hv.y;
        const float r2 = d3_r2(x, y);
        int i_lo = (int)ceilf(hv.z + cw.x);
        if (i_lo < 0) i_lo += nphi;
        if (i_lo >= nphi) i_lo -= nphi;                  // (u is finite and in [-1/2, n_phi - 1/2): stage.cu; |lo| < n_phi)

        // dilated association: (entry >> 1) above ~column (equal votes and |dj| in two columns: the smaller linear
        // bin wins, D8)
        typename EntryT<TILE32>::pkey_t bestp = 0;

        if (!(hm_c > 0.0f)) {
            // ---- exact D3 sequence at every column of the window: classes without a usable bound ----
            if (active) walk_exact_window<MODE, TILE32>(c, d, a, tl, sidx, i_lo, steps, cols);
        } else {
            // ---- fast path: the lane's window, two columns at a time ----
            const float r2Ak = __fmaf_rn(r2, fk.A_f, fk.d0sqA);
            // first column (even, tile-relative) and number of column pairs of the lane's part of the tile
            int start, my_n, np_total;
            if (FULLPHI) {
                start = i_lo & ~1;                       // one column early when i_lo is odd; never past the window + 2
                if (!active) start = (2 * lane) % nphi;  // lanes without work walk rows of their own (no same-word adds)
                my_n = active ? ((steps + 2) & ~1) : 0;
                np_total = (steps + 2) >> 1;             // the same for every hit of a class
            } else {
                int rel = i_lo - c0;
                if (rel < 0) rel += nphi;
                int n;
                if (rel < cols) { start = rel; n = min(steps, cols - rel); }
                else { const int over = rel + steps - nphi; start = 0; n = over > 0 ? min(over, cols) : 0; }
                if (!active) { start = 0; n = 0; }
                const int se = start & ~1;
                my_n = n > 0 ? n + (start - se) : 0;
                start = se;
                np_total = __reduce_max_sync(0xffffffffu, (my_n + 1) >> 1);
            }
            // lanes without work: every evaluation lands in guard slot 0 and none is ever "uncertain"
            const unsigned hmax_l = active ? (unsigned)nq + 2u + dump : 0u;
            const float hm_l = active ? hm_c : __int_as_float(0x7f800000);
            const f32x2 r2Ak2 = pk2(r2Ak, r2Ak);
            int col = start;
            int rem = my_n;                              // columns left in the lane's part (slab tiles)
            for (int p0 = 0; p0 < np_total; p0 += WALK_CHUNK_PAIRS) {
                const int np = min(WALK_CHUNK_PAIRS, np_total - p0);
                if (FULLPHI && col >= nphi) col -= nphi;
                if (!FULLPHI && rem <= 0) col = 0;       // a finished lane idles at the first pair (table bounds)
                const int col_chunk = col, rem_chunk = rem;
                WRec wr = wrec_init(c, x, y, c0 + col);   // (w, d) of the chunk's first pair, from the cos/sin table
                unsigned rowaddr = tile_saddr + (TILE32 ? (unsigned)col * stride4 : (unsigned)(col >> 1) * stride4);
                const int wrap_t = FULLPHI ? ((nphi - col) >> 1) : 0x7fffffff;   // pair of the chunk at which the lane wraps
                unsigned cinv = EntryT<TILE32>::CINV0 - (unsigned)col;   // association: ~(running tile column of the pair)
                unsigned slowmask = 0u;                  // bit t: pair t of the chunk is uncertain
                // One column pair.  Slot min(h, nq + 2 + dump) of the column's row (results outside [-1, nq] land in a dump
                // slot) -- no range test.  A pair with an uncertain column is flagged and does nothing here (predicated
                // votes / no probe): the redo decides both of its columns with the exact D3 sequence.
                auto pair_step = [&](auto wrap_c, int t, unsigned bit) {
                    constexpr bool WRAP = decltype(wrap_c)::value;
                    const f32x2 th2 = wrec_th(wr.w2, ntd0A2, r2Ak2, nqs2, d0cq2, c0h2);       // t~ - 1/2
                    wrec_step(wr, nkap2);                                                     // the next pair's w
                    const f32x2 yb2 = add2(th2, magic2);
                    const f32x2 dl2 = sub2(th2, add2(yb2, nmagic2));                          // (t~ - 1/2) - J
                    float ybA, ybB, dA, dB;
                    upk2(yb2, ybA, ybB);
                    upk2(dl2, dA, dB);
                    // uncertain: t~ within m of a bin edge, J <= t_D3 < J + 1 not proven (NaN never compares true)
                    bool uns;
                    if (FULLPHI) {
                        uns = fmaxf(fabsf(dA), fabsf(dB)) >= hm_l;
                    } else {                             // slab tiles: the lane's own part of the tile only
                        uns = (fabsf(dA) >= hm_l && rem > 0) || (fabsf(dB) >= hm_l && rem > 1);
                    }
                    // a flagged pair is sent to guard slot 0 of its rows (never flushed, empty in association tiles): the
                    // redo decides both of its columns
                    const unsigned hcap = (MODE == WALK_VOTE && uns) ? 0u : hmax_l;     // (association: the probe result is dropped instead)
                    const unsigned hA = min((unsigned)(__float_as_int(ybA) - (WALK_MAGIC_BITS - 1)), hcap);   // slot J + 1
                    const unsigned hB = min((unsigned)(__float_as_int(ybB) - (WALK_MAGIC_BITS - 1)), hcap);
                    unsigned adA = addr_w(rowaddr, hA), adB = addr_w(TILE32 ? rowaddr + stride4 : rowaddr, hB);
                    if (!FULLPHI) {
                        adA = rem > 0 ? adA : trash_saddr;  adB = rem > 1 ? adB : trash_saddr;   // rows past the tile: scratch word
                        rem -= 2;
                    }
                    HOUGH_CHECK((adA >= tile_saddr && adA + 4u <= tile_alloc_end) || adA == trash_saddr);
                    HOUGH_CHECK((adB >= tile_saddr && adB + 4u <= tile_alloc_end) || adB == trash_saddr);
                    if (MODE == WALK_VOTE) {
                        red_shared(adA, 1u);
                        red_shared(adB, TILE32 ? 1u : 65536u);
                    } else {
                        // best (entry >> 1, ~column) of the lane; the q/pT bin and the entry's sign bit are recovered
                        // after the loop by re-evaluating the winning column (fast_bin_direct)
                        const unsigned entA = TILE32 ? lds_u32(adA) : lds_u16(adA);
                        const unsigned entB = TILE32 ? lds_u32(adB) : lds_u16(adB + 2u);
                        const typename EntryT<TILE32>::pkey_t pA = EntryT<TILE32>::pkey_inv(entA, cinv);
                        const typename EntryT<TILE32>::pkey_t pB = EntryT<TILE32>::pkey_inv(entB, cinv - 1u);
                        const typename EntryT<TILE32>::pkey_t pm = pA > pB ? pA : pB;      // ties: the smaller column
                        if (!uns && pm > bestp) bestp = pm;      // flagged pairs are probed by the redo
                        cinv -= 2u;
                    }
                    if (uns) slowmask |= bit;
                    rowaddr += TILE32 ? 2u * stride4 : stride4;
                    if (WRAP && rowaddr >= tile_end) { rowaddr -= tile_bytes; cinv += (unsigned)nphi; }   // past column n_phi - 1
                    (void)t;
                };
                // a chunk in groups of four pairs (constant flag bits inside a group), then the tail; WRAP: some lane of
                // the warp passes column n_phi - 1 inside the chunk (warp-uniform choice of the compiled variant)
                auto run_chunk = [&](auto wrap_c) {
                    int t = 0;
#pragma unroll 1
                    for (; t + 4 <= np; t += 4) {
                        unsigned m4 = slowmask;
                        slowmask = 0u;
                        pair_step(wrap_c, t, 1u);
                        pair_step(wrap_c, t + 1, 2u);
                        pair_step(wrap_c, t + 2, 4u);
                        pair_step(wrap_c, t + 3, 8u);
                        slowmask = m4 | (slowmask << t);
                    }
#pragma unroll 1
                    for (; t < np; ++t) {
                        unsigned m4 = slowmask;
                        slowmask = 0u;
                        pair_step(wrap_c, t, 1u);
                        slowmask = m4 | (slowmask << t);
                    }
                };
                if (FULLPHI && __any_sync(0xffffffffu, wrap_t < np)) run_chunk(std::true_type{});
                else run_chunk(std::false_type{});
                col += 2 * np;                           // FULLPHI: reduced modulo n_phi at the top of the next chunk
                // uncertain pairs of the chunk -> the warp's redo queue, one round per set bit: slots dealt by ballot, the
                // queue drained 32 entries at a time by the whole warp; entries that do not fit 32 bits: redone on the spot
                // (a prefix sum over the lanes' flag counts was measured slower than these rounds)
                unsigned any = __ballot_sync(0xffffffffu, slowmask != 0u);
                int wq_n = WS_SMEM ? (any != 0u ? ws[2] : 0) : wqn_r;
                const bool had_any = any != 0u;
                while (any != 0u) {
                    if (slowmask != 0u) {
                        const int t = __ffs(slowmask) - 1;
                        slowmask &= slowmask - 1u;
                        int cc = col_chunk + 2 * t;
                        if (FULLPHI && cc >= nphi) cc -= nphi;
                        unsigned live = 3u;
                        if (!FULLPHI) live = (rem_chunk - 2 * t > 0 ? 1u : 0u) | (rem_chunk - 2 * t > 1 ? 2u : 0u);
                        HOUGH_CHECK(!wq_ok || (wq_n >= 0 && wq_n + __popc(any & lt) < WALK_WQ_CAP));
                        HOUGH_CHECK(cc >= 0 && cc < slab_cols && (cc & 1) == 0);
                        if (wq_ok) wq[wq_n + __popc(any & lt)] = wq_pack(sidx - ev_begin, cc, live);
                        else walk_redo_pair<MODE, TILE32>(c, d, a, tl, sidx, cc, live);
                    }
                    if (wq_ok) {
                        wq_n += __popc(any);
                        if (wq_n >= 32) {
                            wq_n -= 32;
                            walk_drain<MODE, TILE32>(c, d, a, tl, wq + wq_n, 32, ev_begin, lane);
                        }
                    }
                    any = __ballot_sync(0xffffffffu, slowmask != 0u);
                }
                if (WS_SMEM) {
                    if (had_any) { __syncwarp(); if (lane == 0) ws[2] = wq_n; __syncwarp(); }
                } else {
                    wqn_r = wq_n;
                }
            }
        }
        if (MODE == WALK_ASSIGN) {
            const unsigned eh = EntryT<TILE32>::ent_hi(bestp);          // entry >> 1: votes + 1 above (15 - |dj|)
            if (eh >> 4) {
                // the winning column's bin again (an unflagged pair: the fast slot IS the D3 bin), then the full entry
                const float4 hw = hv;
                const int bcol = EntryT<TILE32>::col_of(bestp);
                const float2 T = __ldg(c.cs + c0 + bcol);
                int J;
                if (!fast_bin_direct(fk, hw.x, hw.y, __fmaf_rn(r2, fk.A_f, fk.d0sqA), T, hm_c, J))
                    J = d3_exact_bin(hw.x, hw.y, r2, T.x, T.y, d.x, d.y, d.z, c.A_f, c.qmin, c.inv_wq, c.nq_f, c.model != 0);
                const unsigned ent = tile_entry<TILE32>(s_tile, stride, bcol, J);
                const int adj = 15 - (int)((ent >> 1) & 15u);
                const int jc = J + ((ent & 1u) ? -adj : adj);
                atomicMax(a.best_key + __float_as_int(hw.w), walk_key((ent >> 5) - 1u, adj, row_lin0 + (unsigned)(bcol * nq + jc)));
            }
        }
    }
    __syncwarp();
    {
        const int wq_n = WS_SMEM ? ws[2] : wqn_r;
        if (wq_n > 0) walk_drain<MODE, TILE32>(c, d, a, tl, wq, wq_n, ev_begin, lane);
    }
    if (MODE == WALK_ASSIGN) return;
    __syncthreads();

    // ---- flush: the tile is written to the global accumulator exactly once (A3); guard slots are dropped ----
    const size_t row0 = ((size_t)e * c.n_d0 + k) * (size_t)nphi + c0;      // first global row of the tile
    if (TILE32 && OUT16) {
        unsigned short* g = reinterpret_cast<unsigned short*>(a.accum) + row0 * nq;
        for (int ci = warp; ci < cols; ci += WALK_WARPS)
            for (int j = lane; j < nq; j += 32) g[(size_t)ci * nq + j] = (unsigned short)s_tile[ci * stride + j + 1];
    } else if (TILE32) {
        int* g = reinterpret_cast<int*>(a.accum) + row0 * nq;
        for (int ci = warp; ci < cols; ci += WALK_WARPS)
            for (int j = lane; j < nq; j += 32) g[(size_t)ci * nq + j] = (int)s_tile[ci * stride + j + 1];
    } else if (OUT16) {
        if ((nq & 1) == 0) {                             // two bins per 32-bit store; a pair row feeds both of its columns
            uint32_t* g = reinterpret_cast<uint32_t*>(reinterpret_cast<unsigned short*>(a.accum) + row0 * nq);
            const int rw = nq >> 1;
            for (int pr = warp; pr < (cols >> 1); pr += WALK_WARPS) {
                const uint32_t* trow = s_tile + pr * stride + 1;
                uint32_t* gA = g + (size_t)(2 * pr) * rw;
                for (int jw = lane; jw < rw; jw += 32) {
                    const uint32_t w0 = trow[2 * jw], w1 = trow[2 * jw + 1];
                    gA[jw] = __byte_perm(w0, w1, 0x5410u);
                    gA[rw + jw] = __byte_perm(w0, w1, 0x7632u);
                }
            }
        } else {
            unsigned short* g = reinterpret_cast<unsigned short*>(a.accum) + row0 * nq;
            for (int ci = warp; ci < cols; ci += WALK_WARPS)
                for (int j = lane; j < nq; j += 32)
                    g[(size_t)ci * nq + j] = (unsigned short)((s_tile[(ci >> 1) * stride + j + 1] >> (16 * (ci & 1))) & 0xffffu);
        }
    } else {
        int* g = reinterpret_cast<int*>(a.accum) + row0 * nq;
        for (int ci = warp; ci < cols; ci += WALK_WARPS)
            for (int j = lane; j < nq; j += 32)
                g[(size_t)ci * nq + j] = (int)((s_tile[(ci >> 1) * stride + j + 1] >> (16 * (ci & 1))) & 0xffffu);
    }
}

// tile shape of a call: as many columns as fit the shared-memory budget, then split further until the grid
// fills the GPU; slab widths are even (column pairs)
inline void walk_shape(const hough_plan* p, int n_events, int& n_slabs, int& slab_cols) {
    const int nphi = p->c.n_phi;
    n_slabs = (nphi + p->tile_max_cols - 1) / p->tile_max_cols;
#ifdef HOUGH_CHECKS
    { const char* es = getenv("HOUGH_FORCE_SLABS"); if (es && atoi(es) > n_slabs) n_slabs = atoi(es); }   // checks build only
#endif
    const long long want = 3LL * p->sm_count;
    while ((long long)n_slabs * p->c.n_d0 * n_events < want && (nphi + n_slabs - 1) / n_slabs > 32) n_slabs *= 2;
    slab_cols = (nphi + n_slabs - 1) / n_slabs;
    slab_cols += slab_cols & 1;
    n_slabs = (nphi + slab_cols - 1) / slab_cols;
}

template <int MODE, bool TILE32, bool OUT16, bool FULLPHI>
int walk_launch(hough_plan* p, int n_events, WalkArgs a, cudaStream_t st) {
    const size_t smem = walk_smem_bytes(a.slab_cols, a.stride, TILE32, p->c.n_class, FULLPHI);
    auto kern = walk_kernel<MODE, TILE32, OUT16, FULLPHI>;
    // opt-in shared memory is a per-device function attribute: one cached size per (instantiation, device), raised
    // only when a call needs more (benign if two host threads race: both set a sufficient value)
    static size_t smem_configured[HOUGH_MAX_DEVICES] = {};
    const int dev = p->device >= 0 && p->device < HOUGH_MAX_DEVICES ? p->device : 0;
    if (smem > smem_configured[dev] || p->device >= HOUGH_MAX_DEVICES) {
        HOUGH_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        smem_configured[dev] = smem;
    }
    const long long grid = (long long)a.n_slabs * p->c.n_d0 * n_events;
    if (grid > 0x7fffffffLL) return HOUGH_ERR_UNSUPPORTED;
    a.exact_only = p->exact_walk;
    a.m_scale = p->m_scale;
    kern<<<(unsigned)grid, walk_threads(MODE), smem, st>>>(p->c, a);
    HOUGH_CUDA_TRY(cudaGetLastError());
    hough_count_launches(1);
    return HOUGH_OK;
}

template <int MODE>
int walk_dispatch(hough_plan* p, int n_events, WalkArgs a, bool tile32, bool out16, cudaStream_t st) {
    const bool full = a.n_slabs == 1;
    if (tile32 && out16 && MODE == WALK_VOTE)
        return full ? walk_launch<MODE, true, true, true>(p, n_events, a, st)
                    : walk_launch<MODE, true, true, false>(p, n_events, a, st);
    if (tile32)
        return full ? walk_launch<MODE, true, false, true>(p, n_events, a, st)
                    : walk_launch<MODE, true, false, false>(p, n_events, a, st);
    if (out16 && MODE == WALK_VOTE)
        return full ? walk_launch<MODE, false, true, true>(p, n_events, a, st)
                    : walk_launch<MODE, false, true, false>(p, n_events, a, st);
    return full ? walk_launch<MODE, false, false, true>(p, n_events, a, st)
                : walk_launch<MODE, false, false, false>(p, n_events, a, st);
}

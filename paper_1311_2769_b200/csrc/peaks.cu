// peaks.cu -- A4: local-maximum search with ordered compaction ("local maxima"; D5-D7).
//
// Tiled path (default): a CTA owns PEAK_BLOCK_BINS consecutive bins of one event (whole phi0 rows of one d0
// slice) and stages those rows, their two phi0 neighbours and the same rows of slices k-1 and k+1 in shared
// memory, so the accumulator is read from L2/HBM with coalesced row copies only.
//   K3a  peak_tile_kernel<EMIT=false> : D5 test from the tile -> per-block count
//   K3b  scan kernels                 : per-event scan of block counts, then scan of event totals -> cand_offsets
//   K3c  peak_tile_kernel<EMIT=true>  : same test, ranks from the scans, records (centroid D7) written in
//                                       ascending (event, k, i, j) order for rank < capacity
// Generic path (a block that spans two d0 slices, or rows too long for the tile): per-bin global loads,
//   peak_mask_kernel (1 bit per bin + per-block count) and peak_emit_kernel (per mask word).
#include <type_traits>

#include "common.cuh"

namespace {

template <bool U16>
__device__ __forceinline__ int load_bin(const void* __restrict__ acc, size_t idx) {
    if (U16) return (int)__ldg(reinterpret_cast<const unsigned short*>(acc) + idx);
    return __ldg(reinterpret_cast<const int*>(acc) + idx);
}

// D5: is bin (k,i,j) with value a a peak?  `ev` points at the event's accumulator.
template <bool U16>
__device__ __forceinline__ bool is_peak(const HoughConsts& c, const void* __restrict__ acc, size_t ebase, int k,
                                        int i, int j, int a) {
    const int nphi = c.n_phi, nq = c.n_qpt, nd = c.n_d0;
    bool peak = true;
#pragma unroll
    for (int dk = -1; dk <= 1; ++dk) {
        const int kk = k + dk;
        if (kk < 0 || kk >= nd) continue;
#pragma unroll
        for (int di = -1; di <= 1; ++di) {
            int ii = i + di;
            ii = ii < 0 ? ii + nphi : (ii >= nphi ? ii - nphi : ii);
            const size_t row = ebase + ((size_t)kk * nphi + ii) * nq;
#pragma unroll
            for (int dj = -1; dj <= 1; ++dj) {
                const int jj = j + dj;
                if (jj < 0 || jj >= nq) continue;
                if (dk == 0 && di == 0 && dj == 0) continue;
                const int v = load_bin<U16>(acc, row + jj);
                const bool before = dk < 0 || (dk == 0 && (di < 0 || (di == 0 && dj < 0)));
                peak = peak && (before ? (a > v) : (a >= v));
            }
        }
    }
    return peak;
}

template <bool U16>
__global__ void __launch_bounds__(256) peak_mask_kernel(HoughConsts c, const void* __restrict__ acc, int threshold,
                                                        int blocks_per_event, uint32_t* __restrict__ mask,
                                                        int32_t* __restrict__ block_cnt) {
    const int e = blockIdx.y, blk = blockIdx.x;
    const size_t ebase = (size_t)e * (size_t)c.bins_per_event;
    const int row_bins = c.n_phi * c.n_qpt;
    int cnt = 0;
    for (int it = 0; it < PEAK_BLOCK_BINS / 256; ++it) {
        const int b = blk * PEAK_BLOCK_BINS + it * 256 + threadIdx.x;
        bool pk = false;
        if (b < c.bins_per_event) {
            const int a = load_bin<U16>(acc, ebase + b);
            if (a >= threshold) {
                const int k = b / row_bins;
                const int r = b - k * row_bins;
                const int i = r / c.n_qpt;
                const int j = r - i * c.n_qpt;
                pk = is_peak<U16>(c, acc, ebase, k, i, j, a);
            }
        }
        const unsigned m = __ballot_sync(0xffffffffu, pk);
        if ((threadIdx.x & 31) == 0) {
            const int word = b >> 5;
            if (word < c.words_per_event) mask[(size_t)e * c.words_per_event + word] = m;
            cnt += __popc(m);
        }
    }
    __shared__ int s_cnt[8];
    if ((threadIdx.x & 31) == 0) s_cnt[threadIdx.x >> 5] = cnt;
    __syncthreads();
    if (threadIdx.x == 0) {
        int t = 0;
        for (int w = 0; w < 8; ++w) t += s_cnt[w];
        block_cnt[(size_t)e * blocks_per_event + blk] = t;
    }
}

__global__ void __launch_bounds__(1024) scan_blocks_kernel(int32_t* block_cnt, int blocks_per_event,
                                                           int32_t* event_cnt) {
    const int e = blockIdx.x;
    cta_exclusive_scan(block_cnt + (size_t)e * blocks_per_event, blocks_per_event, event_cnt + e);
}

__global__ void __launch_bounds__(1024) scan_events_kernel(int32_t* event_cnt, int n_events,
                                                           int32_t* __restrict__ cand_offsets) {
    __shared__ int32_t total;
    cta_exclusive_scan(event_cnt, n_events, &total);
    __syncthreads();
    for (int e = threadIdx.x; e < n_events; e += 1024) cand_offsets[e] = event_cnt[e];
    if (threadIdx.x == 0) cand_offsets[n_events] = total;
}

// One CTA = one peak block (PEAK_BLOCK_BINS bins = 128 mask words).  The block's candidates are dealt to the threads
// by rank (thread t takes candidates t, t + 128, ...), so the lanes of a warp stay busy however the peaks cluster.
template <bool U16>
__global__ void __launch_bounds__(128) peak_emit_kernel(HoughConsts c, const void* __restrict__ acc,
                                                        int blocks_per_event, const uint32_t* __restrict__ mask,
                                                        const int32_t* __restrict__ block_off,
                                                        const int32_t* __restrict__ cand_offsets,
                                                        hough_candidate* __restrict__ cands, int capacity,
                                                        int32_t* __restrict__ word_rank) {
    typedef typename std::conditional<U16, int, long long>::type mom_t;     // 27 * 65535 fits an int
    __shared__ uint32_t s_mask[PEAK_BLOCK_BINS / 32];
    __shared__ int s_pref[PEAK_BLOCK_BINS / 32 + 1];
    __shared__ int s_w[4];
    const int e = blockIdx.y, blk = blockIdx.x;
    const int word = blk * (PEAK_BLOCK_BINS / 32) + threadIdx.x;
    const bool valid = word < c.words_per_event;
    const uint32_t m = valid ? mask[(size_t)e * c.words_per_event + word] : 0u;
    // CTA exclusive scan of popc(m) over 128 threads
    const int v = __popc(m);
    int x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, x, o);
        if ((threadIdx.x & 31) >= o) x += y;
    }
    if ((threadIdx.x & 31) == 31) s_w[threadIdx.x >> 5] = x;
    __syncthreads();
    int prefix = x - v;
    for (int w = 0; w < (int)(threadIdx.x >> 5); ++w) prefix += s_w[w];
    const int base = cand_offsets[e] + block_off[(size_t)e * blocks_per_event + blk];
    if (valid && word_rank) word_rank[(size_t)e * c.words_per_event + word] = base + prefix;
    s_mask[threadIdx.x] = m;
    s_pref[threadIdx.x] = prefix;
    const int total = s_w[0] + s_w[1] + s_w[2] + s_w[3];
    if (threadIdx.x == 0) s_pref[PEAK_BLOCK_BINS / 32] = total;
    __syncthreads();

    const size_t ebase = (size_t)e * (size_t)c.bins_per_event;
    const int nphi = c.n_phi, nq = c.n_qpt, nd = c.n_d0;
    const int row_bins = nphi * nq;
    for (int ci = threadIdx.x; ci < total; ci += 128) {
        const int rank = base + ci;
        if (rank >= capacity) break;                     // ranks ascend with ci
        int lo = 0, hi = PEAK_BLOCK_BINS / 32;           // last word with s_pref[word] <= ci
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (s_pref[mid] <= ci) lo = mid; else hi = mid;
        }
        uint32_t mm = s_mask[lo];
        for (int skip = ci - s_pref[lo]; skip > 0; --skip) mm &= mm - 1;
        const int b = (blk * (PEAK_BLOCK_BINS / 32) + lo) * 32 + (__ffs(mm) - 1);
        const int k = b / row_bins;
        const int r = b - k * row_bins;
        const int i = r / nq;
        const int j = r - i * nq;
        mom_t S = 0, Sj = 0, Si = 0, Sk = 0;
        int a = 0;
#pragma unroll
        for (int dk = -1; dk <= 1; ++dk) {
            const int kk = k + dk;
            if (kk < 0 || kk >= nd) continue;
#pragma unroll
            for (int di = -1; di <= 1; ++di) {
                int ii = i + di;
                ii = ii < 0 ? ii + nphi : (ii >= nphi ? ii - nphi : ii);
                const size_t row = ebase + ((size_t)kk * nphi + ii) * nq + j;
                // the row's three bins at once (missing q/pT neighbours count 0): row sum and left-right difference
                const int vL = j > 0 ? load_bin<U16>(acc, row - 1) : 0;
                const int vC = load_bin<U16>(acc, row);
                const int vR = j + 1 < nq ? load_bin<U16>(acc, row + 1) : 0;
                const mom_t rs = (mom_t)vL + vC + vR;
                S += rs; Sj += (mom_t)(vR - vL);
                if (di > 0) Si += rs; else if (di < 0) Si -= rs;
                if (dk > 0) Sk += rs; else if (dk < 0) Sk -= rs;
                if (dk == 0 && di == 0) a = vC;
            }
        }
        hough_write_candidate(c, cands + rank, e, k, i, j, a, (long long)S, (long long)Sj, (long long)Si, (long long)Sk);
    }
}


// ---- tiled path ------------------------------------------------------------------------------------------
template <bool U16> struct BinT { typedef int type; };
template <> struct BinT<true> { typedef unsigned short type; };

// shared-memory bytes of the halo tile of one block: 3 slices x (rows + 2) x n_qpt bins
inline size_t peak_tile_bytes(const HoughConsts& c) {
    const size_t rows = (size_t)(PEAK_BLOCK_BINS + c.n_qpt - 1) / c.n_qpt + 1;      // rows a block can touch
    return 3 * (rows + 2) * (size_t)c.n_qpt * (c.is_u16 ? 2 : 4) + 16;
}

// A block that spans two d0 slices (n_phi * n_qpt not a multiple of PEAK_BLOCK_BINS): per-bin global loads.
template <bool U16, bool EMIT>
__device__ void peak_block_generic(const HoughConsts& c, const void* __restrict__ acc, int threshold, int e, int blk,
                                   int blocks_per_event, int32_t* __restrict__ block_cnt,
                                   const int32_t* __restrict__ cand_offsets, hough_candidate* __restrict__ cands,
                                   int capacity, int* s_warp_cnt) {
    const int nphi = c.n_phi, nq = c.n_qpt, nd = c.n_d0;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const size_t ebase = (size_t)e * (size_t)c.bins_per_event;
    int base = 0;
    if (EMIT) base = cand_offsets[e] + block_cnt[(size_t)e * blocks_per_event + blk];
    int cnt = 0;
    for (int it = 0; it < PEAK_BLOCK_BINS / 256; ++it) {
        const int b = blk * PEAK_BLOCK_BINS + it * 256 + tid;
        bool pk = false;
        int a = 0, k = 0, i = 0, j = 0;
        if (b < c.bins_per_event) {
            const int r = b / nq;
            j = b - r * nq;
            k = r / nphi;
            i = r - k * nphi;
            a = load_bin<U16>(acc, ebase + b);
            if (a >= threshold) pk = is_peak<U16>(c, acc, ebase, k, i, j, a);
        }
        const unsigned m = __ballot_sync(0xffffffffu, pk);
        if (!EMIT) {
            if (lane == 0) cnt += __popc(m);
            continue;
        }
        if (lane == 0) s_warp_cnt[warp] = __popc(m);
        __syncthreads();
        int before_me = 0, total = 0;
        for (int w = 0; w < 8; ++w) {
            const int n = s_warp_cnt[w];
            if (w < warp) before_me += n;
            total += n;
        }
        const int rank = base + before_me + __popc(m & ((1u << lane) - 1u));
        if (pk && rank < capacity) {
            long long S = 0, Sj = 0, Si = 0, Sk = 0;
            for (int dk = -1; dk <= 1; ++dk) {
                const int kk = k + dk;
                if (kk < 0 || kk >= nd) continue;
                for (int di = -1; di <= 1; ++di) {
                    int ii = i + di;
                    ii = ii < 0 ? ii + nphi : (ii >= nphi ? ii - nphi : ii);
                    for (int dj = -1; dj <= 1; ++dj) {
                        const int jj = j + dj;
                        if (jj < 0 || jj >= nq) continue;
                        const int v = load_bin<U16>(acc, ebase + ((size_t)kk * nphi + ii) * nq + jj);
                        S += v; Sj += (long long)v * dj; Si += (long long)v * di; Sk += (long long)v * dk;
                    }
                }
            }
            hough_write_candidate(c, cands + rank, e, k, i, j, a, S, Sj, Si, Sk);
        }
        base += total;
        __syncthreads();
    }
    if (!EMIT) {
        if (lane == 0) s_warp_cnt[warp] = cnt;
        __syncthreads();
        if (tid == 0) {
            int t = 0;
            for (int w = 0; w < 8; ++w) t += s_warp_cnt[w];
            block_cnt[(size_t)e * blocks_per_event + blk] = t;
        }
    }
}

constexpr int PEAK_WARP_BINS = PEAK_BLOCK_BINS / 8;     // consecutive bins owned by one warp of the block

template <bool U16, bool EMIT>
__global__ void __launch_bounds__(256) peak_tile_kernel(HoughConsts c, const void* __restrict__ acc, int threshold,
                                                        int blocks_per_event, int32_t* __restrict__ block_cnt,
                                                        const int32_t* __restrict__ cand_offsets,
                                                        hough_candidate* __restrict__ cands, int capacity) {
    typedef typename BinT<U16>::type bin_t;
    extern __shared__ __align__(16) unsigned char peak_smem[];
    __shared__ int s_warp_cnt[8];
    __shared__ unsigned short s_list[8][PEAK_WARP_BINS];
    bin_t* tile = reinterpret_cast<bin_t*>(peak_smem);
    const int e = blockIdx.y, blk = blockIdx.x;
    const int nphi = c.n_phi, nq = c.n_qpt, nd = c.n_d0;
    const int b0 = blk * PEAK_BLOCK_BINS;
    const int b1 = min(b0 + PEAK_BLOCK_BINS, c.bins_per_event);
    const int r_a = b0 / nq, r_b = (b1 - 1) / nq;          // global rows (k * n_phi + i) touched by the block
    const int k = r_a / nphi;
    if ((r_b / nphi) != k) {
        peak_block_generic<U16, EMIT>(c, acc, threshold, e, blk, blocks_per_event, block_cnt, cand_offsets, cands, capacity,
                                      s_warp_cnt);
        return;
    }
    const int i_a = r_a - k * nphi;
    const int tr = (r_b - r_a + 1) + 2;                     // tile rows per slice: i_a - 1 .. i_a + n_rows
    const bin_t* ev = reinterpret_cast<const bin_t*>(acc) + (size_t)e * (size_t)c.bins_per_event;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // ---- stage the halo tile: slices k-1, k, k+1 (rows of absent slices are never read) ----
    {
        const bool vec = ((nq * (int)sizeof(bin_t)) % 16 == 0) && ((reinterpret_cast<uintptr_t>(ev) & 15u) == 0);
        for (int s = 0; s < 3; ++s) {
            const int kk = k + s - 1;
            if (kk < 0 || kk >= nd) continue;
            if (vec) {
                const int v_per_row = nq * (int)sizeof(bin_t) / 16;
                for (int rr = warp; rr < tr; rr += 8) {
                    int ii = i_a - 1 + rr;
                    ii = ii < 0 ? ii + nphi : (ii >= nphi ? ii - nphi : ii);
                    const uint4* src = reinterpret_cast<const uint4*>(ev + ((size_t)kk * nphi + ii) * nq);
                    uint4* dst = reinterpret_cast<uint4*>(tile + ((size_t)s * tr + rr) * nq);
                    for (int vv = lane; vv < v_per_row; vv += 32) dst[vv] = __ldg(src + vv);
                }
            } else {
                for (int rr = warp; rr < tr; rr += 8) {
                    int ii = i_a - 1 + rr;
                    ii = ii < 0 ? ii + nphi : (ii >= nphi ? ii - nphi : ii);
                    const bin_t* src = ev + ((size_t)kk * nphi + ii) * nq;
                    bin_t* dst = tile + ((size_t)s * tr + rr) * nq;
                    for (int jj = lane; jj < nq; jj += 32) dst[jj] = __ldg(src + jj);
                }
            }
        }
    }
    __syncthreads();

    // ---- phase A: each warp compacts the bins of its chunk that reach the threshold (order preserved) ----
    // bin b of the block sits at tile[centre0 + (b - r_a * nq)] (the centre slice's rows are contiguous)
    const int centre0 = (tr + 1) * nq - r_a * nq;
    const int slice_stride = tr * nq;
    const int wb0 = b0 + warp * PEAK_WARP_BINS;
    unsigned short* list = s_list[warp];
    int n = 0;
#pragma unroll 4
    for (int it = 0; it < PEAK_WARP_BINS / 32; ++it) {
        const int off = it * 32 + lane;
        const int b = wb0 + off;
        const bool pass = b < b1 && (int)tile[centre0 + b] >= threshold;
        const unsigned m = __ballot_sync(0xffffffffu, pass);
        if (pass) list[n + __popc(m & ((1u << lane) - 1u))] = (unsigned short)off;
        n += __popc(m);
    }
    __syncwarp();

    // ---- phase B: D5 test of the compacted bins, 32 at a time; survivors are compacted in place ----
    int np = 0;
    for (int base = 0; base < n; base += 32) {
        const int idx = base + lane;
        const bool valid = idx < n;
        const int off = valid ? (int)list[idx] : 0;
        __syncwarp();
        bool pk = false;
        if (valid) {
            const int b = wb0 + off;
            const int ci = centre0 + b;
            const int j = (b - r_a * nq) % nq;
            const int a = (int)tile[ci];
            const bool jlo = j > 0, jhi = j + 1 < nq;
            pk = true;
#pragma unroll
            for (int dk = -1; dk <= 1; ++dk) {
                if (k + dk < 0 || k + dk >= nd) continue;
#pragma unroll
                for (int di = -1; di <= 1; ++di) {
                    const bin_t* row = tile + ci + dk * slice_stride + di * nq;
                    const bool before_row = dk < 0 || (dk == 0 && di < 0);
                    const bool after_row = dk > 0 || (dk == 0 && di > 0);
                    if (jlo) { const int v = (int)row[-1]; pk = pk && ((before_row || !after_row) ? (a > v) : (a >= v)); }
                    if (dk != 0 || di != 0) { const int v = (int)row[0]; pk = pk && (before_row ? (a > v) : (a >= v)); }
                    if (jhi) { const int v = (int)row[1]; pk = pk && (before_row ? (a > v) : (a >= v)); }
                }
            }
        }
        const unsigned m = __ballot_sync(0xffffffffu, pk);
        if (pk) list[np + __popc(m & ((1u << lane) - 1u))] = (unsigned short)off;
        np += __popc(m);
    }
    if (lane == 0) s_warp_cnt[warp] = np;
    __syncthreads();
    if (!EMIT) {
        if (tid == 0) {
            int t = 0;
            for (int w = 0; w < 8; ++w) t += s_warp_cnt[w];
            block_cnt[(size_t)e * blocks_per_event + blk] = t;
        }
        return;
    }

    // ---- phase C (EMIT): ranks in linear-bin order = warps in order, list order inside a warp ----
    int rank0 = cand_offsets[e] + block_cnt[(size_t)e * blocks_per_event + blk];
    for (int w = 0; w < warp; ++w) rank0 += s_warp_cnt[w];
    for (int idx = lane; idx < np; idx += 32) {
        const int rank = rank0 + idx;
        if (rank >= capacity) break;
        const int b = wb0 + (int)list[idx];
        const int ci = centre0 + b;
        const int r = b / nq;
        const int j = b - r * nq;
        const int i = r - k * nphi;
        long long S = 0, Sj = 0, Si = 0, Sk = 0;
#pragma unroll
        for (int dk = -1; dk <= 1; ++dk) {
            if (k + dk < 0 || k + dk >= nd) continue;
#pragma unroll
            for (int di = -1; di <= 1; ++di) {
                const bin_t* row = tile + ci + dk * slice_stride + di * nq;
#pragma unroll
                for (int dj = -1; dj <= 1; ++dj) {
                    if (j + dj < 0 || j + dj >= nq) continue;
                    const int v = (int)row[dj];
                    S += v; Sj += (long long)v * dj; Si += (long long)v * di; Sk += (long long)v * dk;
                }
            }
        }
        hough_write_candidate(c, cands + rank, e, k, i, j, (int)tile[ci], S, Sj, Si, Sk);
    }
}


// ---- slice-walk mask kernel (default when rows are 16-byte multiples) -------------------------------------------
// One thread owns VEC consecutive q/pT bins of one phi0 row (one 16-byte load: 8 uint16 or 4 int32 bins) and walks
// a run of d0 slices k0..k1-1, keeping in registers the rows i-1, i, i+1 of the centre slice, the same rows of the
// next slice and the column maximum of the previous slice.  With
//     V_s[j]  = max over di of slice s           (all of slice k-1 is "before" the centre, all of slice k+1 "after")
//     B[j]    = max(V_{k-1}[j], R_k[i-1][j]),    A[j] = max(V_{k+1}[j], R_k[i+1][j])
// the D5 predicate of bin (k, i, j) with value a is
//     a >= threshold  &&  a > max(B[j-1], B[j], B[j+1], R_k[i][j-1])  &&  a >= max(A[j-1], A[j], A[j+1], R_k[i][j+1]).
// Missing neighbours (q/pT and d0 faces) enter as MISSING = a value below every bin, which leaves both
// comparisons true, i.e. skips them (D5).  The accumulator is read once from L2/HBM per slice run plus a
// one-slice halo at each end of a run; neighbouring rows come from L1.
// Output: the peak bitmask (1 bit per bin) and the per-block peak counts consumed by scan + peak_emit_kernel.
template <bool U16> struct KW { static constexpr int VEC = 4; static constexpr int MISSING = (int)0x80000000; };
template <> struct KW<true> { static constexpr int VEC = 8; static constexpr int MISSING = -1; };

template <bool U16>
__device__ __forceinline__ void kw_load_row(const void* __restrict__ acc, size_t row_bin0, int j0, int nq, bool present,
                                            int (&v)[KW<U16>::VEC + 2]) {
    constexpr int VEC = KW<U16>::VEC;
    constexpr int MISSING = KW<U16>::MISSING;
    if (!present) {
#pragma unroll
        for (int x = 0; x < VEC + 2; ++x) v[x] = MISSING;
        return;
    }
    if (U16) {
        const unsigned short* row = reinterpret_cast<const unsigned short*>(acc) + row_bin0;
        const uint4 q = __ldg(reinterpret_cast<const uint4*>(row + j0));
        v[1] = (int)(q.x & 0xffffu); v[2] = (int)(q.x >> 16);
        v[3] = (int)(q.y & 0xffffu); v[4] = (int)(q.y >> 16);
        v[5] = (int)(q.z & 0xffffu); v[6] = (int)(q.z >> 16);
        v[7] = (int)(q.w & 0xffffu); v[8] = (int)(q.w >> 16);
        v[0] = j0 > 0 ? (int)__ldg(row + j0 - 1) : MISSING;
        v[VEC + 1] = j0 + VEC < nq ? (int)__ldg(row + j0 + VEC) : MISSING;
    } else {
        const int* row = reinterpret_cast<const int*>(acc) + row_bin0;
        const int4 q = __ldg(reinterpret_cast<const int4*>(row + j0));
        v[1] = q.x; v[2] = q.y; v[3] = q.z; v[4] = q.w;
        v[0] = j0 > 0 ? __ldg(row + j0 - 1) : MISSING;
        v[VEC + 1] = j0 + VEC < nq ? __ldg(row + j0 + VEC) : MISSING;
    }
}

__device__ __forceinline__ int kw_max3(int a, int b, int c) { return max(max(a, b), c); }

template <bool U16>
__global__ void __launch_bounds__(256, 2) peak_kwalk_kernel(HoughConsts c, const void* __restrict__ acc, int threshold,
                                                            int n_events, int kseg, int n_seg, int blocks_per_event,
                                                            uint32_t* __restrict__ mask, int32_t* __restrict__ block_cnt) {
    constexpr int VEC = KW<U16>::VEC;
    constexpr int W = VEC + 2;
    const int nphi = c.n_phi, nq = c.n_qpt, nd = c.n_d0;
    const int cpr = nq / VEC;                                   // chunks per row
    const long long strips_per_seg = (long long)nphi * cpr;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = strips_per_seg * n_seg * n_events;
    const bool live = gid < total;                              // (nphi * cpr) % 32 == 0: a warp is all live or all dead
    if (!live) return;
    const int chunk = (int)(gid % cpr);
    const int i = (int)((gid / cpr) % nphi);
    const int seg = (int)((gid / strips_per_seg) % n_seg);
    const int e = (int)(gid / (strips_per_seg * n_seg));
    const int j0 = chunk * VEC;
    const int k0 = seg * kseg, k1 = min(k0 + kseg, nd);
    const int im = i == 0 ? nphi - 1 : i - 1, ip = i == nphi - 1 ? 0 : i + 1;
    const size_t ebin = (size_t)e * (size_t)c.bins_per_event;
    const size_t slice_bins = (size_t)nphi * nq;
    const size_t rm = ebin + (size_t)im * nq, r0 = ebin + (size_t)i * nq, rp = ebin + (size_t)ip * nq;
    unsigned char* mask_bytes = reinterpret_cast<unsigned char*>(mask + (size_t)e * c.words_per_event);

    int Vm[W], Rm[W], R0[W], Rp[W];
    {
        int a[W], b[W], d[W];
        const bool has = k0 > 0;
        const size_t so = (size_t)(has ? k0 - 1 : 0) * slice_bins;
        kw_load_row<U16>(acc, rm + so, j0, nq, has, a);
        kw_load_row<U16>(acc, r0 + so, j0, nq, has, b);
        kw_load_row<U16>(acc, rp + so, j0, nq, has, d);
#pragma unroll
        for (int x = 0; x < W; ++x) Vm[x] = kw_max3(a[x], b[x], d[x]);
        const size_t sc = (size_t)k0 * slice_bins;
        kw_load_row<U16>(acc, rm + sc, j0, nq, true, Rm);
        kw_load_row<U16>(acc, r0 + sc, j0, nq, true, R0);
        kw_load_row<U16>(acc, rp + sc, j0, nq, true, Rp);
    }
    for (int k = k0; k < k1; ++k) {
        int Nm[W], N0[W], Np[W];
        const bool has = k + 1 < nd;
        const size_t sn = (size_t)(has ? k + 1 : k) * slice_bins;
        kw_load_row<U16>(acc, rm + sn, j0, nq, has, Nm);
        kw_load_row<U16>(acc, r0 + sn, j0, nq, has, N0);
        kw_load_row<U16>(acc, rp + sn, j0, nq, has, Np);
        int B[W], A[W];
#pragma unroll
        for (int x = 0; x < W; ++x) {
            B[x] = max(Vm[x], Rm[x]);
            A[x] = max(kw_max3(Nm[x], N0[x], Np[x]), Rp[x]);
        }
        unsigned flags = 0u;
#pragma unroll
        for (int x = 1; x <= VEC; ++x) {
            const int a = R0[x];
            const int before = max(kw_max3(B[x - 1], B[x], B[x + 1]), R0[x - 1]);
            const int after = max(kw_max3(A[x - 1], A[x], A[x + 1]), R0[x + 1]);
            if (a >= threshold && a > before && a >= after) flags |= 1u << (x - 1);
        }
        // bitmask: bin b of the event -> bit (b & 7) of byte (b >> 3)
        const size_t bin0 = ((size_t)k * nphi + i) * nq + j0;
        if (U16) {
            mask_bytes[bin0 >> 3] = (unsigned char)flags;
        } else {
            const unsigned other = __shfl_xor_sync(0xffffffffu, flags, 1);
            if ((threadIdx.x & 1) == 0) mask_bytes[bin0 >> 3] = (unsigned char)(flags | (other << 4));
        }
        // a warp covers 32 * VEC consecutive bins of one slice, i.e. one peak block
        const int cnt = __reduce_add_sync(0xffffffffu, __popc(flags));
        if ((threadIdx.x & 31) == 0 && cnt)
            atomicAdd(block_cnt + (size_t)e * blocks_per_event + (int)(bin0 / PEAK_BLOCK_BINS), cnt);
#pragma unroll
        for (int x = 0; x < W; ++x) {
            Vm[x] = kw_max3(Rm[x], R0[x], Rp[x]);
            Rm[x] = Nm[x]; R0[x] = N0[x]; Rp[x] = Np[x];
        }
    }
}

// ---- packed slice walk for 16-bit bins (threshold in [1, 65535]) ---------------------------------------------------
// Same walk and the same D5 algebra as peak_kwalk_kernel, but the 8 bins of a thread stay packed two per register and
// the maxima / comparisons are the DPX instructions VIMNMX3.U16x2 and VIMNMX.U16x2 (with predicate outputs).  A row is
// 6 words X[0..5]: X[1..4] = the 8 bins, X[0].hi = bin j0 - 1, X[5].lo = bin j0 + 8.  Missing neighbours (q/pT and d0
// faces) enter as 0: with a >= threshold >= 1 both "a > 0" and "a >= 0" hold, i.e. the comparison is skipped (D5).
struct Row6 { unsigned x[6]; };

__device__ __forceinline__ Row6 k16_load_row(const unsigned short* __restrict__ row, int j0, int nq, bool present) {
    Row6 r;
    if (!present) {
#pragma unroll
        for (int w = 0; w < 6; ++w) r.x[w] = 0u;
        return r;
    }
    const uint4 q = __ldg(reinterpret_cast<const uint4*>(row + j0));
    r.x[1] = q.x; r.x[2] = q.y; r.x[3] = q.z; r.x[4] = q.w;
    r.x[0] = j0 > 0 ? ((unsigned)__ldg(row + j0 - 1) << 16) : 0u;
    r.x[5] = j0 + 8 < nq ? (unsigned)__ldg(row + j0 + 8) : 0u;
    return r;
}

__device__ __forceinline__ Row6 k16_max3(const Row6& a, const Row6& b, const Row6& c) {
    Row6 r;
#pragma unroll
    for (int w = 0; w < 6; ++w) r.x[w] = __vimax3_u16x2(a.x[w], b.x[w], c.x[w]);
    return r;
}

__device__ __forceinline__ Row6 k16_max2(const Row6& a, const Row6& b) {
    Row6 r;
#pragma unroll
    for (int w = 0; w < 6; ++w) r.x[w] = __vmaxu2(a.x[w], b.x[w]);
    return r;
}

__global__ void __launch_bounds__(256, 2) peak_kwalk16_kernel(HoughConsts c, const unsigned short* __restrict__ acc,
                                                              int threshold, int n_events, int kseg, int n_seg,
                                                              int blocks_per_event, uint32_t* __restrict__ mask,
                                                              int32_t* __restrict__ block_cnt) {
    const int nphi = c.n_phi, nq = c.n_qpt, nd = c.n_d0;
    const int cpr = nq / 8;                                     // chunks per row
    const long long strips_per_seg = (long long)nphi * cpr;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = strips_per_seg * n_seg * n_events;
    if (gid >= total) return;                                   // (nphi * cpr) % 32 == 0: a warp is all live or all dead
    const int chunk = (int)(gid % cpr);
    const int i = (int)((gid / cpr) % nphi);
    const int seg = (int)((gid / strips_per_seg) % n_seg);
    const int e = (int)(gid / (strips_per_seg * n_seg));
    const int j0 = chunk * 8;
    const int k0 = seg * kseg, k1 = min(k0 + kseg, nd);
    const int im = i == 0 ? nphi - 1 : i - 1, ip = i == nphi - 1 ? 0 : i + 1;
    const size_t slice_bins = (size_t)nphi * nq;
    const unsigned short* ev = acc + (size_t)e * (size_t)c.bins_per_event;
    const unsigned short* pm = ev + (size_t)im * nq;
    const unsigned short* p0 = ev + (size_t)i * nq;
    const unsigned short* pp = ev + (size_t)ip * nq;
    unsigned char* mask_bytes = reinterpret_cast<unsigned char*>(mask + (size_t)e * c.words_per_event);
    const unsigned thr2 = (unsigned)threshold * 0x00010001u;

    // the rows of slice k + 1 are in registers and those of slice k + 2 are in flight while slice k is evaluated
    Row6 Vm, Rm, R0, Rp, Nm, N0, Np;
    {
        const bool has = k0 > 0;
        const size_t so = (size_t)(has ? k0 - 1 : 0) * slice_bins;
        Vm = k16_max3(k16_load_row(pm + so, j0, nq, has), k16_load_row(p0 + so, j0, nq, has), k16_load_row(pp + so, j0, nq, has));
        const size_t sc = (size_t)k0 * slice_bins;
        Rm = k16_load_row(pm + sc, j0, nq, true);
        R0 = k16_load_row(p0 + sc, j0, nq, true);
        Rp = k16_load_row(pp + sc, j0, nq, true);
        const bool has1 = k0 + 1 < nd;
        const size_t s1 = (size_t)(has1 ? k0 + 1 : k0) * slice_bins;
        Nm = k16_load_row(pm + s1, j0, nq, has1);
        N0 = k16_load_row(p0 + s1, j0, nq, has1);
        Np = k16_load_row(pp + s1, j0, nq, has1);
    }
#pragma unroll 3
    for (int k = k0; k < k1; ++k) {
        const bool has2 = k + 2 < nd && k + 1 < k1;              // slice k + 2 is needed only if slice k + 1 is evaluated
        const size_t s2 = (size_t)(has2 ? k + 2 : k) * slice_bins;
        const Row6 Pm = k16_load_row(pm + s2, j0, nq, has2);
        const Row6 P0 = k16_load_row(p0 + s2, j0, nq, has2);
        const Row6 Pp = k16_load_row(pp + s2, j0, nq, has2);
        const Row6 B = k16_max2(Vm, Rm);                        // everything "before" the centre row, per q/pT bin
        const Row6 A = k16_max2(k16_max3(Nm, N0, Np), Rp);      // everything "after" it
        // shifted views: s[w] = {hi of x[w], lo of x[w + 1]} = the left neighbours of word w + 1 = the right ones of word w
        unsigned sB[5], sA[5], sR[5];
#pragma unroll
        for (int w = 0; w < 5; ++w) {
            sB[w] = __byte_perm(B.x[w], B.x[w + 1], 0x5432u);
            sA[w] = __byte_perm(A.x[w], A.x[w + 1], 0x5432u);
            sR[w] = __byte_perm(R0.x[w], R0.x[w + 1], 0x5432u);
        }
        unsigned flags = 0u;
#pragma unroll
        for (int w = 1; w <= 4; ++w) {
            const unsigned a = R0.x[w];
            const unsigned before = __vmaxu2(__vimax3_u16x2(sB[w - 1], B.x[w], sB[w]), sR[w - 1]);
            const unsigned after = __vimax3_u16x2(__vimax3_u16x2(sA[w - 1], A.x[w], sA[w]), sR[w], thr2);
            bool ge_hi, ge_lo, le_hi, le_lo;
            (void)__vibmax_u16x2(a, after, &ge_hi, &ge_lo);     // a >= max(after, threshold)
            (void)__vibmax_u16x2(before, a, &le_hi, &le_lo);    // before >= a  (then a is not a strict maximum)
            flags |= (ge_lo && !le_lo ? 1u : 0u) << (2 * (w - 1));
            flags |= (ge_hi && !le_hi ? 1u : 0u) << (2 * (w - 1) + 1);
        }
        // bitmask: bin b of the event -> bit (b & 7) of byte (b >> 3)
        const size_t bin0 = ((size_t)k * nphi + i) * nq + j0;
        mask_bytes[bin0 >> 3] = (unsigned char)flags;
        // a warp covers 256 consecutive bins of one slice, i.e. one peak block
        const int cnt = __reduce_add_sync(0xffffffffu, __popc(flags));
        if ((threadIdx.x & 31) == 0 && cnt)
            atomicAdd(block_cnt + (size_t)e * blocks_per_event + (int)(bin0 / PEAK_BLOCK_BINS), cnt);
        Vm = k16_max3(Rm, R0, Rp);
        Rm = Nm; R0 = N0; Rp = Np;
        Nm = Pm; N0 = P0; Np = Pp;
    }
}

// ---- streamed packed slice walk (16-bit bins): cp.async ring in shared memory ---------------------------------------
// The walk of peak_kwalk16_kernel with the loads decoupled from the registers: a CTA of 256 threads owns R = 256 /
// (n_qpt / 8) consecutive phi0 rows of one event and one run of d0 slices; slice after slice, the R + 2 rows it needs
// (one halo row each side, cyclic) are copied into a ring of PS_STAGES shared-memory stages with cp.async (16 bytes per
// request, whole rows, coalesced), so PS_STAGES - 1 slices are in flight per CTA while one is evaluated.  Bytes in
// flight are bounded by shared memory instead of registers: the accumulator streams in at HBM speed.
constexpr int PS_STAGES = 6;

__device__ __forceinline__ void ps_cp_async16(unsigned saddr, const void* gptr) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(saddr), "l"(gptr) : "memory");
}
__device__ __forceinline__ void ps_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void ps_wait() { asm volatile("cp.async.wait_group %0;" :: "n"(N) : "memory"); }

__device__ __forceinline__ Row6 ps_load_row(const unsigned short* __restrict__ srow, int j0, int nq) {
    Row6 r;
    const uint4 q = *reinterpret_cast<const uint4*>(srow + j0);
    r.x[1] = q.x; r.x[2] = q.y; r.x[3] = q.z; r.x[4] = q.w;
    r.x[0] = j0 > 0 ? ((unsigned)srow[j0 - 1] << 16) : 0u;
    r.x[5] = j0 + 8 < nq ? (unsigned)srow[j0 + 8] : 0u;
    return r;
}

__global__ void __launch_bounds__(256, 3) peak_stream16_kernel(HoughConsts c, const unsigned short* __restrict__ acc,
                                                               int threshold, int kseg, int n_seg, int blocks_per_event,
                                                               uint32_t* __restrict__ mask, int32_t* __restrict__ block_cnt) {
    extern __shared__ __align__(16) unsigned char ps_smem[];
    const int nphi = c.n_phi, nq = c.n_qpt, nd = c.n_d0;
    const int cpr = nq / 8;                                     // 16-byte chunks per row
    const int R = 256 / cpr;                                    // rows per CTA
    const int rb_per_ev = nphi / R;
    const int rb = blockIdx.x % rb_per_ev;
    const int seg = (blockIdx.x / rb_per_ev) % n_seg;
    const int e = blockIdx.x / (rb_per_ev * n_seg);
    const int tid = threadIdx.x;
    const int rl = tid / cpr, chunk = tid - rl * cpr;
    const int j0 = chunk * 8;
    const int i0 = rb * R, i = i0 + rl;
    const int k0 = seg * kseg, k1 = min(k0 + kseg, nd);
    const int stage_halfwords = (R + 2) * nq;
    const unsigned short* ev = acc + (size_t)e * (size_t)c.bins_per_event;
    unsigned short* s_base = reinterpret_cast<unsigned short*>(ps_smem);
    unsigned char* mask_bytes = reinterpret_cast<unsigned char*>(mask + (size_t)e * c.words_per_event);
    const unsigned thr2 = (unsigned)threshold * 0x00010001u;

    // fill stage `stage` with slice v (rows i0 - 1 .. i0 + R, cyclic); slices outside [0, nd) are all "missing" = 0.
    // A thread copies chunk tid and, for tid < 2 * cpr, chunk 256 + tid (the last two rows): offsets fixed per thread.
    const size_t slice_bins = (size_t)nphi * nq;
    int gi_a = i0 - 1 + rl;
    gi_a = gi_a < 0 ? gi_a + nphi : gi_a;
    const unsigned short* src_a = ev + (size_t)gi_a * nq + j0;              // stage row rl
    const int dst_a = rl * nq + j0;
    const bool has_b = tid < 2 * cpr;
    int gi_b = i0 - 1 + R + rl;                                             // stage rows R, R + 1 (rl = 0, 1 here)
    gi_b = gi_b >= nphi ? gi_b - nphi : gi_b;
    const unsigned short* src_b = ev + (size_t)gi_b * nq + j0;
    const int dst_b = (R + rl) * nq + j0;
    const unsigned s_base_saddr = (unsigned)__cvta_generic_to_shared(s_base);
    auto issue = [&](int v, int stage) {
        const int so = stage * stage_halfwords;
        if (v < 0 || v >= nd) {
            *reinterpret_cast<uint4*>(s_base + so + dst_a) = make_uint4(0u, 0u, 0u, 0u);
            if (has_b) *reinterpret_cast<uint4*>(s_base + so + dst_b) = make_uint4(0u, 0u, 0u, 0u);
        } else {
            const size_t go = (size_t)v * slice_bins;
            ps_cp_async16(s_base_saddr + 2u * (unsigned)(so + dst_a), src_a + go);
            if (has_b) ps_cp_async16(s_base_saddr + 2u * (unsigned)(so + dst_b), src_b + go);
        }
        ps_commit();
    };

    const int v_first = k0 - 1, v_last = k1;                    // virtual slices the run needs
    for (int s = 0; s < PS_STAGES; ++s) {
        if (v_first + s <= v_last) issue(v_first + s, s);
        else ps_commit();
    }
    // Two register sets of rows (X, Y) swap roles every slice ("centre" <-> "next"), so no row is ever copied: the loop
    // is unrolled by two with the names exchanged.
    Row6 Vm, Xm, X0, Xp, Ym, Y0, Yp;
#pragma unroll
    for (int w = 0; w < 6; ++w) Vm.x[w] = Xm.x[w] = X0.x[w] = Xp.x[w] = Ym.x[w] = Y0.x[w] = Yp.x[w] = 0u;
    // one slice step: wait for slice v (iteration it), refill the stage freed by the previous step, load its rows into
    // (Nm, N0, Np) and, from the third step on, evaluate the centre slice held in (Rm, R0, Rp)
    int sc = 0, sp = PS_STAGES - 1;                            // ring stage of this step and of the previous one (it % PS_STAGES, kept incrementally)
    auto step = [&](int it, int v, Row6& Rm, Row6& R0, Row6& Rp, Row6& Nm, Row6& N0, Row6& Np) {
        ps_wait<PS_STAGES - 2>();                               // group `it` (slice v) has landed
        __syncthreads();                                        // ... for every thread; the previous stage is free
        if (it >= 1) {
            const int vn = v - 1 + PS_STAGES;
            if (vn <= v_last) issue(vn, sp);
            else ps_commit();
        }
        const unsigned short* st = s_base + (size_t)sc * stage_halfwords + rl * nq;
        HOUGH_CHECK(sc == it % PS_STAGES && (size_t)(sc * stage_halfwords + (rl + 2) * nq + j0 + 8) * 2 <= (size_t)PS_STAGES * (R + 2) * nq * 2);
        sp = sc;
        sc = sc + 1 == PS_STAGES ? 0 : sc + 1;
        Nm = ps_load_row(st, j0, nq);
        N0 = ps_load_row(st + nq, j0, nq);
        Np = ps_load_row(st + 2 * nq, j0, nq);
        if (it == 0) { Vm = k16_max3(Nm, N0, Np); return; }     // slice k0 - 1: only its column maximum is needed
        if (it == 1) return;                                    // slice k0 becomes the centre of the next step
        const int k = v - 1;                                    // centre slice, k0 <= k < k1
        const Row6 B = k16_max2(Vm, Rm);                        // everything "before" the centre row, per q/pT bin
        const Row6 A = k16_max2(k16_max3(Nm, N0, Np), Rp);      // everything "after" it
        unsigned sB[5], sA[5], sR[5];
#pragma unroll
        for (int w = 0; w < 5; ++w) {
            sB[w] = __byte_perm(B.x[w], B.x[w + 1], 0x5432u);
            sA[w] = __byte_perm(A.x[w], A.x[w + 1], 0x5432u);
            sR[w] = __byte_perm(R0.x[w], R0.x[w + 1], 0x5432u);
        }
        unsigned flags = 0u;
#pragma unroll
        for (int w = 1; w <= 4; ++w) {
            const unsigned a = R0.x[w];
            const unsigned before = __vmaxu2(__vimax3_u16x2(sB[w - 1], B.x[w], sB[w]), sR[w - 1]);
            const unsigned after = __vimax3_u16x2(__vimax3_u16x2(sA[w - 1], A.x[w], sA[w]), sR[w], thr2);
            bool ge_hi, ge_lo, le_hi, le_lo;
            (void)__vibmax_u16x2(a, after, &ge_hi, &ge_lo);     // a >= max(after, threshold)
            (void)__vibmax_u16x2(before, a, &le_hi, &le_lo);    // before >= a  (then a is not a strict maximum)
            flags |= (ge_lo && !le_lo ? 1u : 0u) << (2 * (w - 1));
            flags |= (ge_hi && !le_hi ? 1u : 0u) << (2 * (w - 1) + 1);
        }
        const size_t bin0 = ((size_t)k * nphi + i) * nq + j0;
        HOUGH_CHECK(k >= 0 && k < nd && i >= 0 && i < nphi && bin0 + 8 <= (size_t)c.bins_per_event);
        mask_bytes[bin0 >> 3] = (unsigned char)flags;
        const int cnt = __reduce_add_sync(0xffffffffu, __popc(flags));     // a warp = 256 consecutive bins of one peak block
        if ((tid & 31) == 0 && cnt)
            atomicAdd(block_cnt + (size_t)e * blocks_per_event + (int)(bin0 / PEAK_BLOCK_BINS), cnt);
        Vm = k16_max3(Rm, R0, Rp);
    };
    // step 0 loads into Y, step 1 into X (the first centre), step 2 evaluates X against Y, step 3 Y against X, ...
    for (int it = 0, v = v_first; v <= v_last; it += 2, v += 2) {
        step(it, v, Xm, X0, Xp, Ym, Y0, Yp);
        if (v + 1 <= v_last) step(it + 1, v + 1, Ym, Y0, Yp, Xm, X0, Xp);
    }
}

}  // namespace

extern "C" int hough_find_peaks(hough_plan* p, const void* d_accum, int32_t n_events, int32_t threshold,
                                hough_candidate* d_cands, int32_t capacity, int32_t* d_cand_offsets,
                                void* cuda_stream) {
    if (!p || !d_accum || !d_cand_offsets) return HOUGH_ERR_INVALID_ARG;
    if (n_events < 0 || n_events > p->max_events || capacity < 0) return HOUGH_ERR_INVALID_ARG;
    if (capacity > 0 && !d_cands) return HOUGH_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(d_cands) & 15u) return HOUGH_ERR_INVALID_ARG;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    if (n_events == 0) {
        HOUGH_CUDA_TRY(cudaMemsetAsync(d_cand_offsets, 0, sizeof(int32_t), st));
        return HOUGH_OK;
    }
    if (n_events > 65535) return HOUGH_ERR_UNSUPPORTED;
    const int bpe = p->peak_blocks_per_event;
    dim3 grid(bpe, n_events);
    const size_t tile_bytes = peak_tile_bytes(p->c);
    const int kw_vec = p->c.is_u16 ? 8 : 4;
    const bool kwalk = !p->fullscan && !p->peaks_tiled && p->c.n_qpt % 8 == 0 &&
                       ((long long)p->c.n_phi * (p->c.n_qpt / kw_vec)) % 32 == 0 && PEAK_BLOCK_BINS % (32 * kw_vec) == 0 &&
                       (reinterpret_cast<uintptr_t>(d_accum) & 15u) == 0;
    const bool tiled = !kwalk && !p->fullscan && tile_bytes <= 100 * 1024;
    if (kwalk) {
        // enough slice runs to fill the GPU, each at least 8 slices long (a run re-reads one halo slice per end)
        const long long strips = (long long)p->c.n_phi * (p->c.n_qpt / kw_vec) * n_events;
        int n_seg = 1;
        while (strips * n_seg < 256LL * 2 * p->sm_count * 2 && (p->c.n_d0 + n_seg) / (n_seg + 1) >= 8) ++n_seg;
        const int kseg = (p->c.n_d0 + n_seg - 1) / n_seg;
        n_seg = (p->c.n_d0 + kseg - 1) / kseg;
        const long long threads = strips * n_seg;
        const long long nblk = (threads + 255) / 256;
        if (nblk > 0x7fffffffLL) return HOUGH_ERR_UNSUPPORTED;
        HOUGH_CUDA_TRY(cudaMemsetAsync(p->d_peak_block_cnt, 0, sizeof(int32_t) * (size_t)n_events * bpe, st));
        const int cpr16 = p->c.n_qpt / 8;
        const bool stream16 = p->c.is_u16 && threshold >= 1 && threshold <= 65535 && !p->peaks_scalar && !p->peaks_regs &&
                              cpr16 <= 128 && 256 % cpr16 == 0 && p->c.n_phi % (256 / cpr16) == 0 &&
                              (size_t)PS_STAGES * (256 / cpr16 + 2) * p->c.n_qpt * 2 <= 64 * 1024;
        if (stream16) {
            const int R = 256 / cpr16;
            const size_t smem = (size_t)PS_STAGES * (R + 2) * p->c.n_qpt * 2;
            static bool configured[HOUGH_MAX_DEVICES] = {};          // per device: the attribute belongs to the device's copy of the function
            const int dev = p->device >= 0 && p->device < HOUGH_MAX_DEVICES ? p->device : 0;
            if (!configured[dev] || p->device >= HOUGH_MAX_DEVICES) {
                HOUGH_CUDA_TRY(cudaFuncSetAttribute(peak_stream16_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024));
                configured[dev] = true;
            }
            const long long nb = (long long)(p->c.n_phi / R) * n_seg * n_events;
            if (nb > 0x7fffffffLL) return HOUGH_ERR_UNSUPPORTED;
            peak_stream16_kernel<<<(unsigned)nb, 256, smem, st>>>(p->c, reinterpret_cast<const unsigned short*>(d_accum), threshold,
                                                                  kseg, n_seg, bpe, p->d_mask, p->d_peak_block_cnt);
        } else if (p->c.is_u16 && threshold >= 1 && threshold <= 65535 && !p->peaks_scalar)
            peak_kwalk16_kernel<<<(unsigned)nblk, 256, 0, st>>>(p->c, reinterpret_cast<const unsigned short*>(d_accum), threshold,
                                                                n_events, kseg, n_seg, bpe, p->d_mask, p->d_peak_block_cnt);
        else if (p->c.is_u16)
            peak_kwalk_kernel<true><<<(unsigned)nblk, 256, 0, st>>>(p->c, d_accum, threshold, n_events, kseg, n_seg, bpe,
                                                                    p->d_mask, p->d_peak_block_cnt);
        else
            peak_kwalk_kernel<false><<<(unsigned)nblk, 256, 0, st>>>(p->c, d_accum, threshold, n_events, kseg, n_seg, bpe,
                                                                     p->d_mask, p->d_peak_block_cnt);
    } else if (tiled) {
        static bool smem_configured_dev[HOUGH_MAX_DEVICES] = {};     // per device; the tiled path never needs more than 100 KB
        const int dev = p->device >= 0 && p->device < HOUGH_MAX_DEVICES ? p->device : 0;
        bool& smem_configured = smem_configured_dev[dev];
        if (!smem_configured || p->device >= HOUGH_MAX_DEVICES) {
            const int cap = 100 * 1024;
            HOUGH_CUDA_TRY(cudaFuncSetAttribute(peak_tile_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap));
            HOUGH_CUDA_TRY(cudaFuncSetAttribute(peak_tile_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap));
            HOUGH_CUDA_TRY(cudaFuncSetAttribute(peak_tile_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap));
            HOUGH_CUDA_TRY(cudaFuncSetAttribute(peak_tile_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap));
            smem_configured = true;
        }
        if (p->c.is_u16) {
            peak_tile_kernel<true, false><<<grid, 256, tile_bytes, st>>>(p->c, d_accum, threshold, bpe, p->d_peak_block_cnt,
                                                                         nullptr, nullptr, 0);
        } else {
            peak_tile_kernel<false, false><<<grid, 256, tile_bytes, st>>>(p->c, d_accum, threshold, bpe, p->d_peak_block_cnt,
                                                                          nullptr, nullptr, 0);
        }
    } else if (p->c.is_u16)
        peak_mask_kernel<true><<<grid, 256, 0, st>>>(p->c, d_accum, threshold, bpe, p->d_mask, p->d_peak_block_cnt);
    else
        peak_mask_kernel<false><<<grid, 256, 0, st>>>(p->c, d_accum, threshold, bpe, p->d_mask, p->d_peak_block_cnt);
    HOUGH_CUDA_TRY(cudaGetLastError());
    scan_blocks_kernel<<<n_events, 1024, 0, st>>>(p->d_peak_block_cnt, bpe, p->d_event_cnt);
    HOUGH_CUDA_TRY(cudaGetLastError());
    scan_events_kernel<<<1, 1024, 0, st>>>(p->d_event_cnt, n_events, d_cand_offsets);
    HOUGH_CUDA_TRY(cudaGetLastError());
    if (tiled) {
        if (p->c.is_u16)
            peak_tile_kernel<true, true><<<grid, 256, tile_bytes, st>>>(p->c, d_accum, threshold, bpe, p->d_peak_block_cnt,
                                                                        d_cand_offsets, d_cands, capacity);
        else
            peak_tile_kernel<false, true><<<grid, 256, tile_bytes, st>>>(p->c, d_accum, threshold, bpe, p->d_peak_block_cnt,
                                                                         d_cand_offsets, d_cands, capacity);
    } else if (p->c.is_u16)
        peak_emit_kernel<true><<<grid, 128, 0, st>>>(p->c, d_accum, bpe, p->d_mask, p->d_peak_block_cnt, d_cand_offsets,
                                                     d_cands, capacity, nullptr);
    else
        peak_emit_kernel<false><<<grid, 128, 0, st>>>(p->c, d_accum, bpe, p->d_mask, p->d_peak_block_cnt, d_cand_offsets,
                                                      d_cands, capacity, nullptr);
    HOUGH_CUDA_TRY(cudaGetLastError());
    hough_count_launches(4);
    return HOUGH_OK;
}

// peaks.cu -- A4: local-maximum search with ordered compaction ("local maxima"; D5-D7).
//
// K3a  peak_mask_kernel : per bin, threshold + 3x3(x3) test -> 1 bit per bin (warp ballot), per-block count
// K3b  scan kernels     : per-event scan of block counts, then scan of event totals -> cand_offsets
// K3c  peak_emit_kernel : per mask word, rank = offsets + popcounts; write records (centroid D7) in
//                         ascending (event, k, i, j) order for rank < capacity
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

template <bool U16>
__global__ void __launch_bounds__(128) peak_emit_kernel(HoughConsts c, const void* __restrict__ acc,
                                                        int blocks_per_event, const uint32_t* __restrict__ mask,
                                                        const int32_t* __restrict__ block_off,
                                                        const int32_t* __restrict__ cand_offsets,
                                                        hough_candidate* __restrict__ cands, int capacity,
                                                        int32_t* __restrict__ word_rank) {
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
    __shared__ int s_w[4];
    if ((threadIdx.x & 31) == 31) s_w[threadIdx.x >> 5] = x;
    __syncthreads();
    int prefix = x - v;
    for (int w = 0; w < (int)(threadIdx.x >> 5); ++w) prefix += s_w[w];
    const int rank0 = cand_offsets[e] + block_off[(size_t)e * blocks_per_event + blk] + prefix;
    if (valid && word_rank) word_rank[(size_t)e * c.words_per_event + word] = rank0;
    if (m == 0u) return;

    const size_t ebase = (size_t)e * (size_t)c.bins_per_event;
    const int nphi = c.n_phi, nq = c.n_qpt, nd = c.n_d0;
    const int row_bins = nphi * nq;
    uint32_t mm = m;
    int rank = rank0;
    while (mm) {
        const int bit = __ffs(mm) - 1;
        mm &= mm - 1;
        if (rank >= capacity) break;
        const int b = word * 32 + bit;
        const int k = b / row_bins;
        const int r = b - k * row_bins;
        const int i = r / nq;
        const int j = r - i * nq;
        long long S = 0, Sj = 0, Si = 0, Sk = 0;
        int a = 0;
        for (int dk = -1; dk <= 1; ++dk) {
            const int kk = k + dk;
            if (kk < 0 || kk >= nd) continue;
            for (int di = -1; di <= 1; ++di) {
                int ii = i + di;
                ii = ii < 0 ? ii + nphi : (ii >= nphi ? ii - nphi : ii);
                const size_t row = ebase + ((size_t)kk * nphi + ii) * nq;
                for (int dj = -1; dj <= 1; ++dj) {
                    const int jj = j + dj;
                    if (jj < 0 || jj >= nq) continue;
                    const int val = load_bin<U16>(acc, row + jj);
                    S += val; Sj += (long long)val * dj; Si += (long long)val * di; Sk += (long long)val * dk;
                    if (dk == 0 && di == 0 && dj == 0) a = val;
                }
            }
        }
        // D7 centroid: every fp32 operation individually rounded
        const float fS = __ll2float_rn(S);
        const float oj = __fdiv_rn(__ll2float_rn(Sj), fS);
        const float oi = __fdiv_rn(__ll2float_rn(Si), fS);
        const float ok = __fdiv_rn(__ll2float_rn(Sk), fS);
        const float tj = __fadd_rn(__fadd_rn((float)j, 0.5f), oj);
        const float qpt = __fadd_rn(c.qpt_min, __fmul_rn(tj, c.wq));
        const float ti = __fadd_rn(__fadd_rn((float)i, 0.5f), oi);
        float ph = __fmul_rn(ti, c.wphi);
        if (ph < 0.0f) ph = __fadd_rn(ph, c.two_pi_f);
        else if (ph >= c.two_pi_f) ph = __fsub_rn(ph, c.two_pi_f);
        float d0 = 0.0f;
        if (nd > 1) {
            const float tk = __fadd_rn(__fadd_rn((float)k, 0.5f), ok);
            d0 = __fadd_rn(c.d0_min, __fmul_rn(tk, c.wd));
        }
        int4* out = reinterpret_cast<int4*>(cands + rank);
        out[0] = make_int4(e, k, i, j);
        out[1] = make_int4(a, __float_as_int(ph), __float_as_int(qpt), __float_as_int(d0));
        ++rank;
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
    if (p->c.is_u16)
        peak_mask_kernel<true><<<grid, 256, 0, st>>>(p->c, d_accum, threshold, bpe, p->d_mask, p->d_peak_block_cnt);
    else
        peak_mask_kernel<false><<<grid, 256, 0, st>>>(p->c, d_accum, threshold, bpe, p->d_mask, p->d_peak_block_cnt);
    HOUGH_CUDA_TRY(cudaGetLastError());
    scan_blocks_kernel<<<n_events, 1024, 0, st>>>(p->d_peak_block_cnt, bpe, p->d_event_cnt);
    HOUGH_CUDA_TRY(cudaGetLastError());
    scan_events_kernel<<<1, 1024, 0, st>>>(p->d_event_cnt, n_events, d_cand_offsets);
    HOUGH_CUDA_TRY(cudaGetLastError());
    if (p->c.is_u16)
        peak_emit_kernel<true><<<grid, 128, 0, st>>>(p->c, d_accum, bpe, p->d_mask, p->d_peak_block_cnt, d_cand_offsets,
                                                     d_cands, capacity, nullptr);
    else
        peak_emit_kernel<false><<<grid, 128, 0, st>>>(p->c, d_accum, bpe, p->d_mask, p->d_peak_block_cnt, d_cand_offsets,
                                                      d_cands, capacity, nullptr);
    HOUGH_CUDA_TRY(cudaGetLastError());
    hough_count_launches(4);
    return HOUGH_OK;
}

// microbench.cu -- K6: peak-rate microbenchmarks for the roofline denominators MEASURED_PEAKS.json lacks
// (shared-memory atomic rate, non-atomic RMW rate, L2/HBM red.add rate, fp32 issue rate of the D3 sequence).
#include <algorithm>

#include "common.cuh"

namespace {

constexpr int MB_THREADS = 256;
constexpr int MB_WORDS = 16384;     // 64 KB tile
constexpr int MB_ITERS = 4096;

__global__ void __launch_bounds__(MB_THREADS) mb_smem_atomic(int mode, unsigned* __restrict__ sink) {
    extern __shared__ unsigned s_tile[];
    for (int i = threadIdx.x; i < MB_WORDS; i += MB_THREADS) s_tile[i] = 0;
    __syncthreads();
    unsigned state = (blockIdx.x * MB_THREADS + threadIdx.x) * 2654435761u + 12345u;
    unsigned idx = threadIdx.x;
    if (mode == 0) {            // conflict-free: a warp touches 32 consecutive words
#pragma unroll 8
        for (int it = 0; it < MB_ITERS; ++it) {
            atomicAdd(&s_tile[idx], 1u);
            idx = (idx + 4128u) & (MB_WORDS - 1);      // 4128 = 129*32: keeps lane->bank mapping
        }
    } else if (mode == 1) {     // random words
#pragma unroll 8
        for (int it = 0; it < MB_ITERS; ++it) {
            state = state * 1664525u + 1013904223u;
            atomicAdd(&s_tile[state >> 18], 1u);
        }
    } else if (mode == 2) {     // non-atomic load + add + store, conflict-free, thread-private words
        volatile unsigned* vt = s_tile;
#pragma unroll 8
        for (int it = 0; it < MB_ITERS; ++it) {
            vt[idx] = vt[idx] + 1u;
            idx = (idx + 4096u + 256u) & (MB_WORDS - 1);   // stays on this thread's residue class mod 256
        }
    } else if (mode == 5) {     // random column in a 128-bin row chosen per warp (same-address collisions)
#pragma unroll 8
        for (int it = 0; it < MB_ITERS; ++it) {
            state = state * 1664525u + 1013904223u;
            const unsigned row = ((threadIdx.x >> 5) * 16u + (it & 15)) * 128u;
            atomicAdd(&s_tile[(row + (state >> 27) * 1u) & (MB_WORDS - 1)], 1u);
        }
    } else if (mode == 6) {     // kind 5's addresses, but the vote of the ODD column of a packed pair word: + 1 << 16
#pragma unroll 8
        for (int it = 0; it < MB_ITERS; ++it) {
            state = state * 1664525u + 1013904223u;
            const unsigned row = ((threadIdx.x >> 5) * 16u + (it & 15)) * 128u;
            atomicAdd(&s_tile[(row + (state >> 27) * 1u) & (MB_WORDS - 1)], 65536u);
        }
    } else if (mode == 7) {     // kind 6 with warp-aggregated adds: __match_any_sync on the word, the leader adds count << 16
#pragma unroll 8
        for (int it = 0; it < MB_ITERS; ++it) {
            state = state * 1664525u + 1013904223u;
            const unsigned row = ((threadIdx.x >> 5) * 16u + (it & 15)) * 128u;
            const unsigned word = (row + (state >> 27) * 1u) & (MB_WORDS - 1);
            const unsigned peers = __match_any_sync(0xffffffffu, word);
            if ((peers & ((1u << (threadIdx.x & 31)) - 1u)) == 0u) atomicAdd(&s_tile[word], (unsigned)__popc(peers) << 16);
        }
    }
    __syncthreads();
    unsigned acc = 0;
    for (int i = threadIdx.x; i < MB_WORDS; i += MB_THREADS) acc += s_tile[i];
    if (acc == 0xFFFFFFFFu) sink[0] = acc;
}

__global__ void __launch_bounds__(MB_THREADS) mb_global_red(unsigned* __restrict__ region, unsigned mask_words) {
    unsigned state = (blockIdx.x * MB_THREADS + threadIdx.x) * 2654435761u + 777u;
#pragma unroll 8
    for (int it = 0; it < 512; ++it) {
        state = state * 1664525u + 1013904223u;
        atomicAdd(region + ((state >> 4) & mask_words), 1u);
    }
}

__global__ void __launch_bounds__(MB_THREADS) mb_d3_rate(HoughConsts c, float r2, unsigned* __restrict__ sink) {
    float w = -50.0f + 0.001f * (float)(blockIdx.x * MB_THREADS + threadIdx.x);
    int acc = 0;
#pragma unroll 4
    for (int it = 0; it < MB_ITERS; ++it) {
        acc += d3_bin_from_w(w, r2, 1.25f, 2.5f, 1.5625f, c.A_f, c.qmin, c.inv_wq, c.nq_f);
        w = __fadd_rn(w, 0.0123f);
    }
    if (acc == 0x7fffffff) sink[0] = (unsigned)acc;
}

}  // namespace

extern "C" int hough_microbench(int32_t kind, size_t region_bytes, int32_t iters, double* ops_per_s,
                                void* cuda_stream) {
    if (!ops_per_s || iters <= 0) return HOUGH_ERR_INVALID_ARG;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    int dev = 0, sms = 0;
    HOUGH_CUDA_TRY(cudaGetDevice(&dev));
    HOUGH_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    unsigned* d_sink = nullptr;
    unsigned* d_region = nullptr;
    HOUGH_CUDA_TRY(cudaMalloc(&d_sink, 64));
    cudaEvent_t e0, e1;
    HOUGH_CUDA_TRY(cudaEventCreate(&e0));
    HOUGH_CUDA_TRY(cudaEventCreate(&e1));
    double ops = 0.0;
    unsigned mask_words = 0;
    const int grid_smem = sms * 3;            // 3 CTAs of 64 KB per SM
    const int grid_glob = sms * 8;
    if (kind == 3) {
        size_t words = 1;
        while (words * 2 * 4 <= region_bytes) words *= 2;
        if (words < 1024) words = 1024;
        mask_words = (unsigned)(words - 1);
        HOUGH_CUDA_TRY(cudaMalloc(&d_region, words * 4));
        HOUGH_CUDA_TRY(cudaMemsetAsync(d_region, 0, words * 4, st));
    }
    if (kind == 0 || kind == 1 || kind == 2 || (kind >= 5 && kind <= 7))
        HOUGH_CUDA_TRY(cudaFuncSetAttribute(mb_smem_atomic, cudaFuncAttributeMaxDynamicSharedMemorySize, MB_WORDS * 4));
    HoughConsts c{};
    c.A_f = 0.0056960564f; c.qmin = -1.0f; c.inv_wq = 64.0f; c.nq_f = 128.0f;
    float best_ms = 1e30f;
    for (int it = 0; it < iters + 1; ++it) {
        HOUGH_CUDA_TRY(cudaEventRecord(e0, st));
        switch (kind) {
            case 0: case 1: case 2: case 5: case 6: case 7:
                mb_smem_atomic<<<grid_smem, MB_THREADS, MB_WORDS * 4, st>>>(kind, d_sink);
                ops = (double)grid_smem * MB_THREADS * MB_ITERS;
                break;
            case 3:
                mb_global_red<<<grid_glob, MB_THREADS, 0, st>>>(d_region, mask_words);
                ops = (double)grid_glob * MB_THREADS * 512;
                break;
            case 4:
                mb_d3_rate<<<sms * 8, MB_THREADS, 0, st>>>(c, 12100.0f, d_sink);
                ops = (double)sms * 8 * MB_THREADS * MB_ITERS;
                break;
            default:
                cudaFree(d_sink); cudaFree(d_region); cudaEventDestroy(e0); cudaEventDestroy(e1);
                return HOUGH_ERR_INVALID_ARG;
        }
        HOUGH_CUDA_TRY(cudaGetLastError());
        HOUGH_CUDA_TRY(cudaEventRecord(e1, st));
        HOUGH_CUDA_TRY(cudaEventSynchronize(e1));
        float ms = 0.f;
        HOUGH_CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
        if (it > 0) best_ms = std::min(best_ms, ms);     // first launch is warm-up
    }
    *ops_per_s = ops / (best_ms * 1e-3);
    cudaFree(d_sink);
    cudaFree(d_region);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return HOUGH_OK;
}

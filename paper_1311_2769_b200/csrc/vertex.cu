// vertex.cu -- second Hough transform: displaced vertices from the found straight tracks ("apply a
// Hough transform to the track maxima"; reading D10).
//
// A vertex at polar position (R, Phi) is on the line (phi0, d0) iff d0 = R sin(Phi - phi0).  Every kept candidate
// (column i, d0 bin j) of a LINE-model track space votes, for every vertex-azimuth column m (the track space's own
// column centres), for the one compatible radius, with the prescribed fp32 sequence (each operation rounded):
//     d  = qmin + ((float)j + 0.5f) * wq                      centre of the candidate's d0 bin
//     sd = sin_m * cos_i - cos_m * sin_i                       sin(Phi_m - phi0_i)
//     R  = d / sd;  t = R * inv_wr;  vote iff 0 <= t < n_r;  vacc[e][m][(int)t] += 1
// The work is tiny (kept displaced tracks x n_phi columns): one CTA per (event, chunk of candidates), threads over
// columns, votes with global red.add into the int32 vertex accumulator [event][n_phi][n_r] (zeroed here).
#include "common.cuh"

namespace {

constexpr int VTX_CANDS_PER_CTA = 64;

__global__ void __launch_bounds__(256) vertex_vote_kernel(HoughConsts c, const hough_candidate* __restrict__ cands,
                                                          const int32_t* __restrict__ cand_off, int capacity,
                                                          const uint8_t* __restrict__ keep, float d_abs_min, int n_r,
                                                          float inv_wr, int32_t* __restrict__ vacc) {
    const int e = blockIdx.y;
    const int c0 = min(cand_off[e], capacity), c1 = min(cand_off[e + 1], capacity);
    const int first = c0 + blockIdx.x * VTX_CANDS_PER_CTA;
    if (first >= c1) return;
    const int last = min(first + VTX_CANDS_PER_CTA, c1);
    const float nr_f = (float)n_r;
    for (int ci = first; ci < last; ++ci) {
        if (keep && !keep[ci]) continue;                                  // uniform over the CTA
        const int4 q = __ldg(reinterpret_cast<const int4*>(cands + ci)); // event, k, i, j
        const float d = __fadd_rn(c.qmin, __fmul_rn(__fadd_rn((float)q.w, 0.5f), c.wq));
        if (!(fabsf(d) >= d_abs_min)) continue;
        const float2 ti = __ldg(c.cs + q.z);                              // {cos_i, sin_i}
        for (int m = threadIdx.x; m < c.n_phi; m += blockDim.x) {
            const float2 tm = __ldg(c.cs + m);
            const float sd = __fsub_rn(__fmul_rn(tm.y, ti.x), __fmul_rn(tm.x, ti.y));
            const float R = __fdiv_rn(d, sd);
            const float t = __fmul_rn(R, inv_wr);
            if (t >= 0.0f && t < nr_f) atomicAdd(vacc + ((size_t)e * c.n_phi + m) * n_r + (int)t, 1);
        }
    }
}

}  // namespace

extern "C" int hough_vertex_vote(hough_plan* p, const hough_candidate* d_cands, const int32_t* d_cand_offsets,
                                 int32_t n_events, int32_t capacity, const uint8_t* d_cand_keep, float d0_abs_min,
                                 int32_t n_r, float r_max, int32_t* d_vertex_accum, void* cuda_stream) {
    if (!p || !d_cand_offsets || !d_vertex_accum) return HOUGH_ERR_INVALID_ARG;
    if (p->b.model != HOUGH_MODEL_LINE) return HOUGH_ERR_INVALID_ARG;
    if (n_events < 0 || n_events > 65535 || capacity < 0 || n_r <= 0 || !(r_max > 0.0f) || !(d0_abs_min >= 0.0f))
        return HOUGH_ERR_INVALID_ARG;
    if (capacity > 0 && !d_cands) return HOUGH_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(d_cands) & 15u) return HOUGH_ERR_INVALID_ARG;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    if (n_events == 0) return HOUGH_OK;
    HOUGH_CUDA_TRY(cudaMemsetAsync(d_vertex_accum, 0, sizeof(int32_t) * (size_t)n_events * p->c.n_phi * n_r, st));
    if (capacity == 0) return HOUGH_OK;
    const float inv_wr = (float)((double)n_r / (double)r_max);
    // the candidate counts live on the device (no host read): enough CTAs for `capacity` candidates per event
    const int chunks = (capacity + VTX_CANDS_PER_CTA - 1) / VTX_CANDS_PER_CTA;
    dim3 grid(chunks, n_events);
    vertex_vote_kernel<<<grid, 256, 0, st>>>(p->c, d_cands, d_cand_offsets, capacity, d_cand_keep, d0_abs_min, n_r, inv_wr,
                                            d_vertex_accum);
    HOUGH_CUDA_TRY(cudaGetLastError());
    hough_count_launches(1);
    return HOUGH_OK;
}

/* hough.h -- C ABI of libhough_b200: Hough-transform track finding (arXiv 1311.2769) on one B200 (sm_100a).
 *
 * The paper states the method in words only (section 3):
 *   "Each possible instance of a feature starts with zero votes in the parameter space, and then, for each
 *    piece of input data, votes are added to the feature instances that would include that input data.
 *    After all input data has been processed ... looking for local maxima in the parameter space.  After
 *    the initial identification, further computations ... confirm the existence of the track."
 * and PAPER.md:45: the two-parameter space finds curved tracks through the origin; curved displaced tracks
 * need three parameters.  BASELINE.json `north_star` (B:L5) fixes the parameters (phi0, signed q/pT, d0),
 * the call names and the bit-exact fp32 contract.  Every formula below is a reading recorded in DESIGN.md
 * ("Readings" D1-D9, taken from SURVEY.md section 8(c)).
 *
 * Conventions
 *   - Every function returns an int status (HOUGH_OK = 0, errors < 0), never throws, never exits.
 *   - Pointers named d_*  are DEVICE pointers owned by the caller (the library never frees them and keeps
 *     none after the call returns).  Pointers named h_* are HOST pointers.  Plain names are host structs.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - Device-side calls only ENQUEUE work on `cuda_stream` and return: no device synchronisation, no
 *     device->host read (they can be captured into a CUDA graph).  A plan owns one workspace, so one plan
 *     serves one stream at a time.
 *   - Host-detectable argument errors return a negative status and enqueue nothing.
 *   - Accumulator layout: accum[event][k (d0)][i (phi0)][j (q/pT)], j fastest, tightly packed, int32_t
 *     (HOUGH_ACC_I32) or uint16_t (HOUGH_ACC_U16).  U16 precondition: no bin exceeds 65535.
 *   - Hit layout: float xy[n_hits][2] in cm, events concatenated; int32 event_offsets[n_events + 1] with
 *     event_offsets[0] = 0, event_offsets[n_events] = n_hits, non-decreasing.  Hit order inside an event is
 *     arbitrary and affects no output.  d_hits_xy must be 8-byte aligned.
 */
#ifndef HOUGH_B200_H_
#define HOUGH_B200_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { HOUGH_OK = 0, HOUGH_ERR_INVALID_ARG = -1, HOUGH_ERR_CUDA = -2, HOUGH_ERR_ALLOC = -3, HOUGH_ERR_UNSUPPORTED = -4,
       HOUGH_ERR_TOO_LARGE = -5 /* a size beyond the fixed limit of a no-allocation entry point */ };
enum { HOUGH_ACC_I32 = 0, HOUGH_ACC_U16 = 1 };
/* Track model = which parameter is solved per (hit, phi0 column).  HELIX: curved tracks, signed q/pT (D3; the space of
 * B:L5).  LINE: straight displaced tracks ("or straight displaced tracks"; zero field): the impact
 * parameter d0 = y cos(phi0) - x sin(phi0) is solved (D3L), n_d0 must be 1, the binned axis j is d0 in cm over
 * [qpt_min, qpt_max) -- the q/pT fields of hough_binning and of hough_candidate then carry d0 -- and bz is ignored. */
enum { HOUGH_MODEL_HELIX = 0, HOUGH_MODEL_LINE = 1 };

/* Parameter-space binning (B:L5; D2).  n_phi % 4 == 0 (quadrant-symmetric trig tables).  n_d0 == 1 is the
 * two-parameter space of PAPER.md:45 (single d0 slice with centre exactly 0; d0_min/d0_max ignored). */
typedef struct {
    int32_t n_phi, n_qpt, n_d0;
    float qpt_min, qpt_max;       /* GeV^-1, half-open [min, max) */
    float d0_min, d0_max;         /* cm */
    int32_t accum_dtype;          /* HOUGH_ACC_I32 | HOUGH_ACC_U16 */
    int32_t model;                /* HOUGH_MODEL_HELIX | HOUGH_MODEL_LINE */
} hough_binning;

/* Detector description.  bz_tesla enters the vote formula (A = K*Bz/2, K = 0.00299792458 GeV/(T cm)).
 * layer_radius_cm (host pointer, copied; may be NULL with n_layers = 0) is used ONLY to size work
 * (radius classes for hit staging); it never changes a result (S19). */
typedef struct {
    float bz_tesla;
    int32_t n_layers;
    const float* layer_radius_cm;
} hough_geometry;

/* Track candidate = local maximum of the accumulator (D5-D7).  32 bytes. */
typedef struct {
    int32_t event, k, i, j;       /* bin indices: d0 slice k, phi0 column i, q/pT bin j */
    int32_t votes;
    float phi0, qpt, d0;          /* integer-moment centroid over the 3x3(x3) neighbourhood (D7) */
} hough_candidate;

typedef struct hough_plan hough_plan;   /* opaque: device tables + workspace */

/* hough_plan_create (B:L5 "hough_plan_create(binning, detector geometry)"; D2).
 * Validates, builds the fp32 tables (cos/sin of the phi0 column centres from libm in double with exact
 * quadrant symmetry, d0 centres, 2*d0, d0^2, A, qmin, n_qpt/(qmax-qmin)), copies them to the current CUDA
 * device and allocates workspace for at most max_hits hits in at most max_events events per call.
 * Errors: INVALID_ARG (null pointers, n_phi % 4, empty ranges, unknown dtype, non-positive sizes),
 * UNSUPPORTED (bins per event > 2^31-1), ALLOC/CUDA.  *out is untouched on error. */
int hough_plan_create(const hough_binning* binning, const hough_geometry* geometry, int32_t max_hits,
                      int32_t max_events, hough_plan** out);
int hough_plan_destroy(hough_plan* plan);

/* Bytes of an accumulator for n_events events with this plan's binning and dtype (0 if plan is NULL). */
size_t hough_accum_bytes(const hough_plan* plan, int32_t n_events);

/* hough_vote ("votes are added to the feature instances that would include that input data"; D3/D4).
 * OVERWRITES d_accum (n_events accumulators) with the votes of exactly these hits: for every hit and every
 * (phi0 column i, d0 slice k) the one compatible q/pT is solved with the prescribed fp32 sequence
 *     r2 = x*x + y*y;  w = y*cos_i - x*sin_i;  f = x*cos_i + y*sin_i;  vote only if f > 0;
 *     num = d0_k - w;  den = (r2 - 2d0_k*w) + d0_k^2;  v = num * (1/(A*den));  t = (v - qmin)*inv_wq;
 *     vote only if 0 <= t < n_qpt;  j = (int)t;  accum[e][k][i][j] += 1
 * (each operation rounded to nearest-even, no FMA contraction, IEEE reciprocal).
 * HOUGH_MODEL_LINE (D3L): same w, f and forward test, then  t = (w - qpt_min)*inv_w;  vote only if 0 <= t < n_qpt;
 * j = (int)t;  accum[e][0][i][j] += 1.
 * Errors: INVALID_ARG (null pointers, n_hits > max_hits, n_events > max_events, negative sizes), CUDA. */
int hough_vote(hough_plan* plan, const float* d_hits_xy, int32_t n_hits, const int32_t* d_event_offsets,
               int32_t n_events, void* d_accum, void* cuda_stream);

/* hough_find_peaks ("looking for local maxima in the parameter space"; D5-D7).
 * A bin is a peak iff a >= threshold and, over its 3x3 (n_d0 == 1) or 3x3x3 neighbourhood (phi0 cyclic,
 * q/pT and d0 clipped), a > b for neighbours at lexicographically smaller offset (dk,di,dj) and a >= b for
 * the others.  Records are written in ascending (event, k, i, j) order for global rank < capacity;
 * d_cand_offsets[n_events + 1] always receives the exclusive scan of the TRUE per-event counts (overflow is
 * not an error: compare d_cand_offsets[n_events] with capacity).  d_cands may be NULL when capacity == 0.
 * Limit: at most 65535 events per call (one grid row per event); more returns UNSUPPORTED -- split the batch. */
int hough_find_peaks(hough_plan* plan, const void* d_accum, int32_t n_events, int32_t threshold,
                     hough_candidate* d_cands, int32_t capacity, int32_t* d_cand_offsets, void* cuda_stream);

/* hough_assign_hits ("further computations ... confirm the existence of the track"; "cleaned to
 * ... eliminate duplicate tracks"; D8/D9).
 * d_hit_to_cand[h] = the candidate of the hit's own event, among those with rank < capacity, whose column
 * (i,k) the hit votes in at a bin jh with |jh - j| <= assoc_dj, maximising (votes, -|jh-j|, -index); -1 if
 * none.  d_cand_nhits[c] = hits whose best candidate is c; d_cand_keep[c] = (nhits >= min_hits); hits of a
 * dropped candidate become -1 (single pass, no re-assignment).  d_cand_nhits / d_cand_keep hold `capacity`
 * entries; entries at or beyond min(total, capacity) are zeroed.  0 <= assoc_dj <= 15. */
int hough_assign_hits(hough_plan* plan, const float* d_hits_xy, int32_t n_hits, const int32_t* d_event_offsets,
                      int32_t n_events, const hough_candidate* d_cands, const int32_t* d_cand_offsets,
                      int32_t capacity, int32_t assoc_dj, int32_t min_hits, int32_t* d_hit_to_cand,
                      int32_t* d_cand_nhits, uint8_t* d_cand_keep, void* cuda_stream);

/* hough_event_run (P:L37 vote -> local maxima -> further computations, for ONE event; "the two-parameter space";
 * P:L55 / Fig. 2: time per event as a function of the number of tracks).
 * Exactly hough_vote + hough_find_peaks + hough_assign_hits for a single event (n_events == 1, d_event_offsets = {0,
 * n_hits} on the device), with the same outputs bit for bit: d_accum (one accumulator, overwritten), d_cands /
 * d_cand_offsets[2], d_hit_to_cand, d_cand_nhits, d_cand_keep (see those calls for layouts and the capacity rule).
 * For a two-parameter space (n_d0 == 1) whose 16-bit tile fits the shared memory of at most 8 SMs and an event of at
 * most 2560 hits (and a work estimate below the measured break-even with the general path, see below), the whole path runs in ONE launch of a thread-block cluster (accumulator slab in shared memory, steps
 * separated by cluster barriers) -- what a latency-bound small event needs; every other case runs the three calls
 * (plan option "event_general" = 1 forces that; "event_cluster" = 1 takes the cluster whenever it fits, ignoring the work
 * estimate hits x longest window <= 160000 that otherwise gates it).  Enqueues on cuda_stream and returns; graph-capturable.
 * d_event_offsets MUST hold {0, n_hits}: the cluster path takes the event as hits [0, n_hits) and does not read the array
 * (no device->host read to validate it), the three calls do read it -- other contents give path-dependent results.
 * A device (or MIG / MPS partition) on which a cluster of that shape cannot be co-scheduled, or a failing cluster launch,
 * silently takes the three calls instead.
 * Errors: INVALID_ARG (null / misaligned pointers, sizes, assoc_dj > 15), UNSUPPORTED, CUDA. */
int hough_event_run(hough_plan* plan, const float* d_hits_xy, int32_t n_hits, const int32_t* d_event_offsets,
                    void* d_accum, int32_t threshold, hough_candidate* d_cands, int32_t capacity,
                    int32_t* d_cand_offsets, int32_t assoc_dj, int32_t min_hits, int32_t* d_hit_to_cand,
                    int32_t* d_cand_nhits, uint8_t* d_cand_keep, void* cuda_stream);

/* hough_reassign_hits ("cleaned to select only the best candidate ... and eliminate duplicate tracks"; "hits in
 * these tracks are then removed, allowing later iterations"; D12 re-assignment rounds).
 * Call after hough_assign_hits with the same hits, offsets, candidates, capacity and assoc_dj, and with ITS outputs in
 * d_hit_to_cand / d_cand_nhits / d_cand_keep.  D12: in round t every hit takes its best candidate (the D8 key of
 * hough_assign_hits) among the candidates still alive, a candidate stays alive iff >= min_hits hits took it; rounds end
 * when none was dropped or after max_rounds.  Round 1 is hough_assign_hits.  A kept candidate can only gain hits in round
 * 2, so the kept set never changes again: round 2 is the fixed point, and this call runs exactly that round for
 * max_rounds >= 2 (max_rounds == 1: returns at once).  Effect: every hit with d_hit_to_cand[h] == -1 gets the best
 * candidate with d_cand_keep != 0 (or stays -1), d_cand_nhits of that candidate is incremented; hits that had a kept
 * candidate, d_cand_nhits of dropped candidates and d_cand_keep are left as they are.
 * Tiled plans take the candidate-centric association over the surviving candidates, which needs an azimuth-interval table
 * per plan.  Build it at set-up with hough_plan_set_option(plan, "prepare_reassign", 1) (one cudaMalloc + device
 * synchronisation); the pipeline option "reassign" does so for its lanes.  Without that, the first call whose stream is NOT
 * under capture builds it; a call on a capturing stream never allocates or synchronises -- while there is no table (not
 * built yet, does not fit, build failed, or plan option "reassign_walk") the call re-walks the vote columns against the
 * surviving candidates, with the same results.
 * Errors: INVALID_ARG (null pointers, sizes, max_rounds < 1), UNSUPPORTED, CUDA. */
int hough_reassign_hits(hough_plan* plan, const float* d_hits_xy, int32_t n_hits, const int32_t* d_event_offsets,
                        int32_t n_events, const hough_candidate* d_cands, const int32_t* d_cand_offsets,
                        int32_t capacity, int32_t assoc_dj, int32_t max_rounds, int32_t* d_hit_to_cand,
                        int32_t* d_cand_nhits, const uint8_t* d_cand_keep, void* cuda_stream);

/* hough_vertex_vote ("apply a Hough transform to the track maxima" -- displaced vertices; D10).
 * `plan` is the HOUGH_MODEL_LINE plan of the TRACK space that produced d_cands.  Every candidate with d_cand_keep[c] != 0
 * (all candidates when d_cand_keep is NULL), rank < capacity and |d| >= d0_abs_min votes, for every vertex-azimuth
 * column m (the plan's own n_phi column centres), for the radius R = d / sin(Phi_m - phi0_i), where d is the centre of the
 * candidate's d0 bin:  d = qpt_min + ((float)j + 0.5f) * w;  sd = sin_m cos_i - cos_m sin_i;  R = d / sd;  t = R * n_r /
 * r_max;  vote iff 0 <= t < n_r  (each fp32 operation rounded, IEEE division).
 * OVERWRITES d_vertex_accum: int32 [n_events][n_phi][n_r], i.e. the layout of an accumulator with binning
 * {n_phi, n_qpt = n_r, n_d0 = 1, qpt range [0, r_max), int32}: its peaks (hough_find_peaks on such a plan) are the vertex
 * candidates (phi0 field = vertex azimuth, qpt field = vertex radius in cm).
 * Errors: INVALID_ARG (null pointers, plan not of the line model, bad sizes, more than 65535 events per call), CUDA. */
int hough_vertex_vote(hough_plan* plan, const hough_candidate* d_cands, const int32_t* d_cand_offsets, int32_t n_events,
                      int32_t capacity, const uint8_t* d_cand_keep, float d0_abs_min, int32_t n_r, float r_max,
                      int32_t* d_vertex_accum, void* cuda_stream);

/* hough_fit_circles ("further computations (e.g., a full Kalman fit) can be performed to confirm the existence
 * of the track and obtain the best measurement of the track parameters"; D11: an algebraic circle fit in double stands in).
 * For every candidate c < min(d_cand_offsets[n_events], capacity) with d_cand_keep[c] != 0 (all when NULL): Kasa fit
 * (minimise sum (x^2 + y^2 + B x + C y + D)^2) of the hits h with d_hit_to_cand[h] == c, then the D1 parameters of the
 * circle, oriented by the candidate's phi0 column: d_fit[c] = {phi0 [rad, 0..2pi), q/pT [1/GeV; 0 when Bz = 0], d0 [cm],
 * radius [cm]}; d_n_fit[c] = hits used, -(hits) when the fit is not ok (< 3 hits, singular, R^2 <= 0), 0 when no hits /
 * dropped / beyond the list (d_fit then zero).  d_work: caller's scratch, 9 doubles per candidate of `capacity`.
 * Moments are summed with double atomics, so results agree with a sequential sum to ~1e-9 relative, not bit for bit. */
typedef struct { double phi0, qpt, d0, radius; } hough_track_fit;
int hough_fit_circles(hough_plan* plan, const float* d_hits_xy, int32_t n_hits, const int32_t* d_hit_to_cand,
                      const hough_candidate* d_cands, const int32_t* d_cand_offsets, int32_t n_events, int32_t capacity,
                      const uint8_t* d_cand_keep, double* d_work, hough_track_fit* d_fit, int32_t* d_n_fit,
                      void* cuda_stream);

/* hough_fit_circles_static -- hough_fit_circles for callers that cannot allocate device memory (same fit: PAPER.md:37, D11).
 * Some users of this library may not call cudaMalloc where they need the fit: an event loop with a fixed time budget per
 * event (a trigger; cudaMalloc / cudaFree take unbounded time and stall the whole device), or a plug-in inside an
 * application whose GPU memory belongs to another memory manager and which is given only its input and output buffers.
 * hough_fit_circles needs scratch from the caller (d_work) and a plan (whose creation allocates); this call needs neither:
 * the moment sums go to a fixed array inside the library image, HOUGH_FIT_STATIC_MAX_CANDIDATES rows of 9 doubles
 * (4.5 MiB), which every GPU that loads the library holds until the process exits.  The call itself allocates and frees
 * nothing: no cudaMalloc, no cudaFree, no library routine that allocates.
 * Arguments: n_phi and bz_tesla are the two plan values the fit uses (number of phi0 columns of the space the candidates
 * come from; Bz in tesla, 0 gives q/pT = 0); all other arguments, outputs, alignment rules and tolerances are those of
 * hough_fit_circles, computed by the same kernels.  Enqueues on cuda_stream and returns.
 * Rules that follow from the shared array:
 *   - capacity > HOUGH_FIT_STATIC_MAX_CANDIDATES returns HOUGH_ERR_TOO_LARGE and enqueues nothing (split the list, or use
 *     hough_fit_circles with your own scratch);
 *   - there is ONE array per GPU, shared by every call and keeping the last call's sums (each call zeroes the rows it
 *     uses first): calls that can run on the GPU at the same time -- other streams, other threads -- race and give wrong
 *     fits; issue them on one stream or order them with events;
 *   - the first call on each GPU also looks up that GPU's copy of the array (cudaGetSymbolAddress, cached per device
 *     afterwards): make one call per device at start-up (capacity >= 1; n_hits = 0 will do), with that device
 *     current, before any stream capture begins.  cuda_stream must belong to the current device.
 * Errors: INVALID_ARG (null / misaligned pointers, negative sizes, n_phi <= 0), TOO_LARGE, CUDA. */
#define HOUGH_FIT_STATIC_MAX_CANDIDATES 65536
int hough_fit_circles_static(int32_t n_phi, float bz_tesla, const float* d_hits_xy, int32_t n_hits,
                             const int32_t* d_hit_to_cand, const hough_candidate* d_cands, const int32_t* d_cand_offsets,
                             int32_t n_events, int32_t capacity, const uint8_t* d_cand_keep, hough_track_fit* d_fit,
                             int32_t* d_n_fit, void* cuda_stream);

/* Plan options (debug / tuning; results never change).  key "fullscan": 1 = evaluate every (hit,i,k) with
 * no windowing and vote straight into global memory (the bisecting path of SURVEY section 5; also read once at
 * plan creation from the environment: HOUGH_DEBUG_FULLSCAN=1).  "exact_walk": 1 = the windowed walk runs the
 * prescribed D3 sequence at every column (no fast path; HOUGH_DEBUG_EXACT_WALK=1).  "peaks_tiled": 1 = halo-tile
 * peak kernels; "peaks_scalar": 1 = the unpacked slice-walk peak kernel also for 16-bit bins, "peaks_regs": 1 = the packed
 * 16-bit walk with rows held in registers instead of the cp.async shared-memory ring.  "reuse_staging": 1 = the caller promises that a hough_assign_hits call whose hit pointer, offsets
 * pointer, sizes and stream equal those of the preceding hough_vote sees unchanged hits, so the staged (sorted)
 * copy of that vote is reused instead of rebuilt.  "prepare_reassign": 1 = build the table of hough_reassign_hits now
 * (allocates and synchronises; always HOUGH_OK -- without a table that call re-walks the columns).
 * Environment (read at plan creation, work sizing only): HOUGH_SECTORS=n phi sectors of the staging sort
 * (default: n_phi clamped to [32, 1024], halved while the plan's key table max_events x classes x sectors exceeds 32 MiB). */
int hough_plan_set_option(hough_plan* plan, const char* key, int32_t value);

/* Batched multi-event pipeline (B:L5 "a batched multi-event path using CUDA streams and graphs"; B:L10).
 * Runs vote -> find_peaks -> assign_hits over HOST buffers: events are cut into tiles of tile_events, tiles
 * are dealt round-robin to n_streams streams, each with its own plan, accumulator and staging buffers; a
 * stream's per-tile sequence (H2D hits, the three calls, D2H of the counts) is stream-captured, the stream's
 * executable CUDA graph is updated in place (cudaGraphExecUpdate: same topology, other sizes) and launched once per
 * tile; a device kernel rebases tile-local event / candidate indices to global ones before the results are copied
 * into the caller's buffers.  The call blocks until all results are in the host buffers.
 * h_hits_xy and the outputs should be pinned (cudaHostAlloc / cudaHostRegister) for the copies to overlap with the
 * kernels; pageable memory works (plain launches, no graphs) but serialises.
 * Environment: HOUGH_PIPELINE_NO_GRAPHS=1 disables graph capture.
 * Outputs (host): h_hit_to_cand[n_hits] (indices are GLOBAL candidate ranks, events concatenated, -1 = none),
 * h_cand_offsets[n_events + 1], h_cands[cand_capacity] (records of rank < cand_capacity),
 * h_cand_nhits / h_cand_keep [cand_capacity].  Per-tile candidate capacity is tile_cand_capacity; a tile
 * that overflows it sets *h_overflowed (results for that tile are truncated as in hough_find_peaks). */
typedef struct hough_pipeline hough_pipeline;
int hough_pipeline_create(const hough_binning* binning, const hough_geometry* geometry, int32_t tile_events,
                          int32_t max_hits_per_tile, int32_t tile_cand_capacity, int32_t n_streams,
                          hough_pipeline** out);
int hough_pipeline_destroy(hough_pipeline* p);
/* Pipeline options.  "kept_only" = 1: only the candidates that survive duplicate removal (D9, cand_keep = 1) are
 * returned -- the tile's kept records are compacted on the device before the copy, h_cand_offsets are the offsets of
 * the KEPT list, h_hit_to_cand indexes it (hits of dropped candidates are -1 as always), h_cand_nhits follows it and
 * h_cand_keep is 1 for every returned candidate; cand_capacity then bounds the kept list.  All the work (vote, peaks,
 * association) is unchanged; only the result transfer shrinks (config 3: 1.0 GB -> 45 MB per 1024 events).
 * "graphs" = 0 / 1: CUDA graph capture off / on.  "reassign" = 1: every tile's association is followed by the D12
 * re-assignment round (hough_reassign_hits), so h_hit_to_cand / h_cand_nhits are the fixed point of the rounds.
 * INVALID_ARG for unknown keys. */
int hough_pipeline_set_option(hough_pipeline* p, const char* key, int32_t value);
int hough_pipeline_run_host(hough_pipeline* p, const float* h_hits_xy, int32_t n_hits,
                            const int32_t* h_event_offsets, int32_t n_events, int32_t threshold,
                            int32_t assoc_dj, int32_t min_hits, int32_t* h_hit_to_cand,
                            int32_t* h_cand_offsets, hough_candidate* h_cands, int32_t cand_capacity,
                            int32_t* h_cand_nhits, uint8_t* h_cand_keep, int32_t* h_overflowed);

/* Work-sizing tables, for inspection and tests (HOST only, no CUDA call; S19: these never change a result).
 * Hits are grouped into radius classes; for (class c, d0 slice k) every column a hit of that class can vote in
 * lies in the run of `steps[c*n_d0+k]` columns starting at ceil(u + lo_off[c*n_d0+k]) (cyclic), where
 * u = phi * n_phi / 2pi - 0.5 is the hit's azimuth in column units.  The kernels evaluate the exact D3
 * sequence at every column of the run, so a run may be too long but must never miss a voting column.
 * edge_r2[c] = lower r^2 edge of class c (class = largest c with edge_r2[c] <= x*x + y*y; the last class is
 * open-ended).  Output arrays may be NULL; capacities: edge_r2 256 floats, lo_off / steps 256 * n_d0 entries. */
int hough_window_table(const hough_binning* binning, const hough_geometry* geometry, int32_t* n_class,
                       float* edge_r2, float* lo_off, int32_t* steps);

/* Measurement support (K6): peak-rate microbenchmarks for the roofline denominators that
 * MEASURED_PEAKS.json lacks.  Each runs `iters` launches on cuda_stream, synchronises, and writes the
 * average operations per second of the best launch to *ops_per_s.  kind:
 *   0 = shared-memory atomicAdd(u32), conflict-free (lane -> distinct bank), all SMs
 *   1 = shared-memory atomicAdd(u32), random addresses in a 64 KB tile
 *   2 = shared-memory load+add+store (non-atomic RMW), conflict-free
 *   3 = global red.add.u32 to random addresses in a region of `region_bytes` (L2- or HBM-resident)
 *   4 = fp32 issue rate of the D3 vote sequence (no memory), evaluations per second
 *   5 = shared-memory atomicAdd(u32), every warp adds to random bins of one 128-bin row (same-address collisions
 *       included): the address pattern closest to the vote walk's
 *   6 = kind 5's addresses with atomicAdd(u32, 1 << 16): the vote of the odd column of a packed 16-bit pair word
 *   7 = kind 6 warp-aggregated: __match_any_sync on the word, one leader adds (lanes << 16)   (B:L5 "warp-aggregated atomics")
 * Errors: INVALID_ARG (unknown kind, iters <= 0, NULL ops_per_s), CUDA. */
int hough_microbench(int32_t kind, size_t region_bytes, int32_t iters, double* ops_per_s, void* cuda_stream);

/* Process-wide number of CUDA kernel launches this library has issued so far (memsets/copies excluded). */
int64_t hough_kernel_launches(void);

const char* hough_status_string(int status);
/* Library build identity: "libhough_b200 <version> sm_100a". */
const char* hough_version(void);

#ifdef __cplusplus
}
#endif
#endif /* HOUGH_B200_H_ */

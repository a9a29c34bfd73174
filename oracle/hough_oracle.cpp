// hough_oracle.cpp -- CPU ORACLE for the Hough track-finding hot path of arXiv 1311.2769.
//
// *** TEST INFRASTRUCTURE ONLY ***  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may load this.  The product (paper_1311_2769_b200/) never does,
// and this file shares no code, header, table or constant generator with the CUDA path.
//
// Plain, slow, single-threaded, obviously-correct restatement of what the path computes:
//   * PAPER.md:37 (section 3): "Each possible instance of a feature starts with zero votes in the
//     parameter space, and then, for each piece of input data, votes are added to the feature
//     instances that would include that input data ... looking for local maxima in the parameter
//     space ... further computations ... confirm the existence of the track".
//   * PAPER.md:45 (section 3): two-parameter space for curved tracks through the origin; curved
//     displaced tracks need three parameters.
//   * BASELINE.json north_star (B:L5): parameters phi0, signed q/pT, d0; one vote per (phi0, d0)
//     column; 3x3(x3) local maximum above a threshold; hit association + duplicate removal; bin
//     indices from one prescribed IEEE fp32 formula (host: -ffp-contract=off).
// The paper prints no formula, so every definition below is a reading recorded in DESIGN.md
// ("Readings", D1-D9 / S1-S20 of SURVEY.md section 8(c)).  Each function names the reading it follows.
//
// There is no windowing, sorting, blocking or fusion here: the vote is a full scan over every
// (hit, phi0 column, d0 slice).  Build: g++ -O2 -ffp-contract=off (no -ffast-math, no -march=native).
//
// Pins (tests/test_oracle_*.py, run with -m "not gpu"): V1 brute force in double from the
// tangent-chord construction, V2 noiseless helix -> its own bin, V3 closed-form vote count,
// V4 linearity/permutation, V5 2-D special case, V6 quarter-turn shift, V7 peak definition on
// constructed volumes, V8 brute-force vs indexed assignment, V12 re-assignment rounds (hand-built shared-hit case,
// rounds = 1 == D9, fixed point == brute force over the kept candidates).  No function here is "parity unpinned".

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

extern "C" {

typedef struct {
    int32_t n_phi, n_qpt, n_d0;
    float qpt_min, qpt_max;   // GeV^-1, half-open [min, max)
    float d0_min, d0_max;     // cm; ignored when n_d0 == 1
    int32_t model;            // 0: curved tracks, solve q/pT (D3);  1: straight displaced tracks, solve d0 (D3L)
} orc_binning;

typedef struct {
    int32_t event, k, i, j, votes;
    float phi0, qpt, d0;
} orc_candidate;              // 32 bytes

}  // extern "C"

namespace {

const double kPi = 3.14159265358979323846;
const double kGeVPerTeslaCm = 0.00299792458;   // pT[GeV] = K * Bz[T] * R[cm]   (D1)

// D2 -- plan constants, double -> fp32.
struct Tables {
    std::vector<float> cosT, sinT;     // [n_phi]  phi0 column centres
    std::vector<float> d0c, td0, d0sq; // [n_d0]
    float A_f, qmin, inv_wq;
    int model;
};

bool valid_binning(const orc_binning* b) {
    return b && b->n_phi > 0 && b->n_phi % 4 == 0 && b->n_qpt > 0 && b->n_d0 > 0 &&
           b->qpt_max > b->qpt_min && (b->n_d0 == 1 || b->d0_max > b->d0_min) &&
           (b->model == 0 || (b->model == 1 && b->n_d0 == 1));
}

Tables make_tables(const orc_binning& b, float bz) {
    Tables t;
    t.A_f = (float)(0.5 * kGeVPerTeslaCm * (double)bz);
    t.model = b.model;
    t.qmin = b.qpt_min;
    t.inv_wq = (float)((double)b.n_qpt / ((double)b.qpt_max - (double)b.qpt_min));
    const int n = b.n_phi, q = n / 4;
    t.cosT.resize(n);
    t.sinT.resize(n);
    for (int i = 0; i < q; ++i) {                    // first quadrant from libm, in double
        const double theta = ((double)i + 0.5) * (2.0 * kPi / (double)n);
        t.cosT[i] = (float)std::cos(theta);
        t.sinT[i] = (float)std::sin(theta);
    }
    for (int i = 0; i + q < n; ++i) {                // other quadrants by exact symmetry (S6)
        t.cosT[i + q] = -t.sinT[i];
        t.sinT[i + q] = t.cosT[i];
    }
    t.d0c.resize(b.n_d0);
    t.td0.resize(b.n_d0);
    t.d0sq.resize(b.n_d0);
    for (int k = 0; k < b.n_d0; ++k) {
        if (b.n_d0 == 1) {
            t.d0c[k] = 0.0f;
        } else {
            t.d0c[k] = (float)((double)b.d0_min +
                               ((double)k + 0.5) * ((double)b.d0_max - (double)b.d0_min) / (double)b.n_d0);
        }
        t.td0[k] = 2.0f * t.d0c[k];
        t.d0sq[k] = t.d0c[k] * t.d0c[k];
    }
    return t;
}

// D3 -- the q/pT bin of hit (x, y, r2) in column (i, k), or -1 when the hit casts no vote there.
// Every fp32 operation is individually rounded (no FMA: -ffp-contract=off), in exactly this order.
inline int vote_bin(const Tables& t, int n_qpt, float x, float y, float r2, int i, int k) {
    const float c = t.cosT[i], s = t.sinT[i];
    const float yc = y * c;
    const float xs = x * s;
    const float w = yc - xs;                 // w = p . n_hat
    const float xc = x * c;
    const float ys = y * s;
    const float f = xc + ys;                 // f = p . t_hat
    if (!(f > 0.0f)) return -1;              // forward branch only (S4)
    if (t.model == 1) {
        // D3L -- straight displaced track ("or straight displaced tracks"): the zero-curvature limit of D1.
        // A straight line with direction phi0 and signed impact parameter d0 passes through p iff d0 = p . n_hat = w
        // (the hits of one point trace the sinusoid d0 = -x sin(phi0) + y cos(phi0)).  The binned axis j
        // is d0 over [qpt_min, qpt_max) cm (the struct's q/pT fields carry the range of the solved parameter).
        const float dw = w - t.qmin;
        const float tl = dw * t.inv_wq;
        if (!(tl >= 0.0f && tl < (float)n_qpt)) return -1;
        return (int)tl;
    }
    const float num = t.d0c[k] - w;
    const float tw = t.td0[k] * w;
    const float d1 = r2 - tw;
    const float den = d1 + t.d0sq[k];
    const float g = t.A_f * den;
    const float rinv = 1.0f / g;             // IEEE-correct reciprocal
    const float v = num * rinv;
    const float dv = v - t.qmin;
    const float tt = dv * t.inv_wq;
    if (!(tt >= 0.0f && tt < (float)n_qpt)) return -1;   // range test; NaN/inf fall out here (S5)
    return (int)tt;                          // tt >= 0: truncation == floor
}

inline float hit_r2(float x, float y) {
    const float xx = x * x;
    const float yy = y * y;
    return xx + yy;
}

// D5 -- offset order: (dk, di, dj) lexicographically below (0,0,0)?
inline bool offset_is_before(int dk, int di, int dj) {
    if (dk != 0) return dk < 0;
    if (di != 0) return di < 0;
    return dj < 0;
}

}  // namespace

extern "C" {

// D2: export the plan constants (for the pins that check table symmetry / exact representability).
// consts = {A_f, qmin, inv_wq}.  Any output pointer may be null.
int orc_tables(const orc_binning* b, float bz, float* cosT, float* sinT, float* d0c, float* td0,
               float* d0sq, float* consts) {
    if (!valid_binning(b)) return -1;
    Tables t = make_tables(*b, bz);
    if (cosT) std::memcpy(cosT, t.cosT.data(), sizeof(float) * b->n_phi);
    if (sinT) std::memcpy(sinT, t.sinT.data(), sizeof(float) * b->n_phi);
    if (d0c) std::memcpy(d0c, t.d0c.data(), sizeof(float) * b->n_d0);
    if (td0) std::memcpy(td0, t.td0.data(), sizeof(float) * b->n_d0);
    if (d0sq) std::memcpy(d0sq, t.d0sq.data(), sizeof(float) * b->n_d0);
    if (consts) { consts[0] = t.A_f; consts[1] = t.qmin; consts[2] = t.inv_wq; }
    return 0;
}

// D3/D4 -- vote.  accum is int32 [n_events][k_hi-k_lo][n_phi][n_qpt] (j fastest), OVERWRITTEN
// ("starts with zero votes").  [k_lo, k_hi) restricts the d0 slices computed; the full
// accumulator is (0, n_d0).  Returns the number of votes cast, or <0 on bad arguments.
long long orc_vote(const orc_binning* b, float bz, const float* hits_xy, int32_t n_hits,
                   const int32_t* event_offsets, int32_t n_events, int32_t k_lo, int32_t k_hi,
                   int32_t* accum) {
    if (!valid_binning(b) || n_hits < 0 || n_events < 0 || !event_offsets || !accum) return -1;
    if (k_lo < 0 || k_hi > b->n_d0 || k_lo >= k_hi) return -1;
    if (n_hits > 0 && !hits_xy) return -1;
    const Tables t = make_tables(*b, bz);
    const int nk = k_hi - k_lo;
    const size_t per_event = (size_t)nk * b->n_phi * b->n_qpt;
    std::memset(accum, 0, sizeof(int32_t) * per_event * (size_t)n_events);
    long long votes = 0;
    for (int e = 0; e < n_events; ++e) {
        int32_t* acc = accum + per_event * (size_t)e;
        for (int h = event_offsets[e]; h < event_offsets[e + 1]; ++h) {
            const float x = hits_xy[2 * (size_t)h], y = hits_xy[2 * (size_t)h + 1];
            const float r2 = hit_r2(x, y);
            for (int i = 0; i < b->n_phi; ++i) {
                for (int k = k_lo; k < k_hi; ++k) {
                    const int j = vote_bin(t, b->n_qpt, x, y, r2, i, k);
                    if (j < 0) continue;
                    acc[((size_t)(k - k_lo) * b->n_phi + i) * b->n_qpt + j] += 1;
                    ++votes;
                }
            }
        }
    }
    return votes;
}

// D3 for sampled columns: rows[s][0..n_qpt) = accumulator column (event, k, i) of sample s,
// computed one by one (full-size parity on sampled outputs).  cols = int32 [n_samples][3] = (e, k, i).
int orc_vote_columns(const orc_binning* b, float bz, const float* hits_xy, int32_t n_hits,
                     const int32_t* event_offsets, int32_t n_events, const int32_t* cols,
                     int32_t n_samples, int32_t* rows) {
    if (!valid_binning(b) || !event_offsets || !cols || !rows) return -1;
    (void)n_hits;
    const Tables t = make_tables(*b, bz);
    std::memset(rows, 0, sizeof(int32_t) * (size_t)n_samples * b->n_qpt);
    for (int s = 0; s < n_samples; ++s) {
        const int e = cols[3 * s], k = cols[3 * s + 1], i = cols[3 * s + 2];
        if (e < 0 || e >= n_events || k < 0 || k >= b->n_d0 || i < 0 || i >= b->n_phi) return -1;
        for (int h = event_offsets[e]; h < event_offsets[e + 1]; ++h) {
            const float x = hits_xy[2 * (size_t)h], y = hits_xy[2 * (size_t)h + 1];
            const int j = vote_bin(t, b->n_qpt, x, y, hit_r2(x, y), i, k);
            if (j >= 0) rows[(size_t)s * b->n_qpt + j] += 1;
        }
    }
    return 0;
}

// D3 per hit: number of (i, k) columns in which hit h votes (the independent counter of pin V3).
int orc_votes_per_hit(const orc_binning* b, float bz, const float* hits_xy, int32_t n_hits,
                      int32_t* votes_per_hit) {
    if (!valid_binning(b) || !votes_per_hit) return -1;
    const Tables t = make_tables(*b, bz);
    for (int h = 0; h < n_hits; ++h) {
        const float x = hits_xy[2 * (size_t)h], y = hits_xy[2 * (size_t)h + 1];
        const float r2 = hit_r2(x, y);
        int n = 0;
        for (int i = 0; i < b->n_phi; ++i)
            for (int k = 0; k < b->n_d0; ++k)
                if (vote_bin(t, b->n_qpt, x, y, r2, i, k) >= 0) ++n;
        votes_per_hit[h] = n;
    }
    return 0;
}

// D5/D6/D7 -- peaks.  accum: int32 [n_events][k_hi-k_lo][n_phi][n_qpt] holding global slices
// [k_lo, k_hi).  Peaks are reported for slices [ko_lo, ko_hi), which requires every EXISTING
// neighbour slice (ko_lo-1 .. ko_hi, clipped to [0, n_d0)) to lie inside [k_lo, k_hi).
// Full volume: k_lo = ko_lo = 0, k_hi = ko_hi = n_d0.
// cand_offsets [n_events+1] = exclusive scan of the TRUE per-event counts; records are written only
// for global rank < capacity (S12).  Returns the total number of peaks, or <0 on bad arguments.
long long orc_find_peaks(const orc_binning* b, const int32_t* accum, int32_t n_events, int32_t k_lo,
                         int32_t k_hi, int32_t ko_lo, int32_t ko_hi, int32_t threshold,
                         orc_candidate* cands, long long capacity, int32_t* cand_offsets) {
    if (!valid_binning(b) || !accum || !cand_offsets || n_events < 0) return -1;
    if (k_lo < 0 || k_hi > b->n_d0 || k_lo >= k_hi || ko_lo < k_lo || ko_hi > k_hi || ko_lo > ko_hi) return -1;
    if (ko_lo < ko_hi) {
        const int need_lo = ko_lo - 1 < 0 ? 0 : ko_lo - 1;
        const int need_hi = ko_hi + 1 > b->n_d0 ? b->n_d0 : ko_hi + 1;
        if (need_lo < k_lo || need_hi > k_hi) return -1;
    }
    const int nphi = b->n_phi, nq = b->n_qpt, nd = b->n_d0;
    const int nk = k_hi - k_lo;
    const size_t per_event = (size_t)nk * nphi * nq;
    const float wq = (float)(((double)b->qpt_max - (double)b->qpt_min) / (double)nq);
    const float wphi = (float)((2.0 * kPi) / (double)nphi);
    const float wd = (float)(((double)b->d0_max - (double)b->d0_min) / (double)nd);
    const float two_pi_f = (float)(2.0 * kPi);
    long long total = 0;
    for (int e = 0; e < n_events; ++e) {
        cand_offsets[e] = (int32_t)total;
        const int32_t* acc = accum + per_event * (size_t)e;
        for (int k = ko_lo; k < ko_hi; ++k)
            for (int i = 0; i < nphi; ++i)
                for (int j = 0; j < nq; ++j) {
                    const int32_t a = acc[((size_t)(k - k_lo) * nphi + i) * nq + j];
                    if (a < threshold) continue;                                   // S9: a >= threshold
                    bool peak = true;
                    long long S = 0, Sj = 0, Si = 0, Sk = 0;
                    for (int dk = -1; dk <= 1 && peak; ++dk) {
                        const int kk = k + dk;
                        if (kk < 0 || kk >= nd) continue;                          // clipped in d0 (S10)
                        for (int di = -1; di <= 1 && peak; ++di) {
                            const int ii = (i + di + nphi) % nphi;                 // phi0 is cyclic (S10)
                            for (int dj = -1; dj <= 1; ++dj) {
                                const int jj = j + dj;
                                if (jj < 0 || jj >= nq) continue;                  // clipped in q/pT
                                const int32_t v = acc[((size_t)(kk - k_lo) * nphi + ii) * nq + jj];
                                S += v; Sj += (long long)v * dj; Si += (long long)v * di; Sk += (long long)v * dk;
                                if (dk == 0 && di == 0 && dj == 0) continue;
                                if (offset_is_before(dk, di, dj)) { if (!(a > v)) { peak = false; break; } }
                                else                              { if (!(a >= v)) { peak = false; break; } }
                            }
                        }
                    }
                    if (!peak) continue;
                    if (cands && total < capacity) {
                        orc_candidate& c = cands[total];
                        c.event = e; c.k = k; c.i = i; c.j = j; c.votes = a;
                        const float fS = (float)S;                                  // D7 centroid
                        const float oj = (float)Sj / fS;
                        const float oi = (float)Si / fS;
                        const float ok = (float)Sk / fS;
                        const float tj = ((float)j + 0.5f) + oj;
                        c.qpt = b->qpt_min + tj * wq;
                        const float ti = ((float)i + 0.5f) + oi;
                        float ph = ti * wphi;
                        if (ph < 0.0f) ph = ph + two_pi_f;
                        else if (ph >= two_pi_f) ph = ph - two_pi_f;
                        c.phi0 = ph;
                        if (nd == 1) {
                            c.d0 = 0.0f;
                        } else {
                            const float tk = ((float)k + 0.5f) + ok;
                            c.d0 = b->d0_min + tk * wd;
                        }
                    }
                    ++total;
                }
    }
    cand_offsets[n_events] = (int32_t)total;
    return total;
}

// D8 key: (votes, -|dj|, -index) lexicographic, as a 64-bit integer.
static inline uint64_t assign_key(int32_t votes, int adj, long long index) {
    return ((uint64_t)(uint32_t)votes << 40) | ((uint64_t)(255 - adj) << 32) |
           (uint64_t)(0xFFFFFFFFu - (uint32_t)index);
}

// D9 applied to a filled hit_to_cand.
static void dedup(int32_t n_hits, long long n_cands, int32_t min_hits, int32_t* hit_to_cand,
                  int32_t* cand_nhits, uint8_t* cand_keep) {
    for (long long c = 0; c < n_cands; ++c) cand_nhits[c] = 0;
    for (int h = 0; h < n_hits; ++h)
        if (hit_to_cand[h] >= 0) cand_nhits[hit_to_cand[h]] += 1;
    for (long long c = 0; c < n_cands; ++c) cand_keep[c] = cand_nhits[c] >= min_hits ? 1 : 0;
    for (int h = 0; h < n_hits; ++h)
        if (hit_to_cand[h] >= 0 && !cand_keep[hit_to_cand[h]]) hit_to_cand[h] = -1;   // no re-assignment
}

// D8/D9 -- brute force over (hit, candidate) pairs.  n_cands = min(total, capacity) records present.
// apply_dedup = 0 returns the raw best candidate per hit (before the min_hits cut).
int orc_assign_brute(const orc_binning* b, float bz, const float* hits_xy, int32_t n_hits,
                     const int32_t* event_offsets, int32_t n_events, const orc_candidate* cands,
                     const int32_t* cand_offsets, long long capacity, int32_t assoc_dj, int32_t min_hits,
                     int32_t apply_dedup, int32_t* hit_to_cand, int32_t* cand_nhits, uint8_t* cand_keep) {
    if (!valid_binning(b) || !event_offsets || !cand_offsets || !hit_to_cand) return -1;
    const Tables t = make_tables(*b, bz);
    for (int e = 0; e < n_events; ++e) {
        long long c0 = cand_offsets[e], c1 = cand_offsets[e + 1];
        if (c1 > capacity) c1 = capacity;
        for (int h = event_offsets[e]; h < event_offsets[e + 1]; ++h) {
            const float x = hits_xy[2 * (size_t)h], y = hits_xy[2 * (size_t)h + 1];
            const float r2 = hit_r2(x, y);
            uint64_t best = 0;
            int32_t best_c = -1;
            for (long long c = c0; c < c1; ++c) {
                const int jh = vote_bin(t, b->n_qpt, x, y, r2, cands[c].i, cands[c].k);
                if (jh < 0) continue;
                const int adj = jh > cands[c].j ? jh - cands[c].j : cands[c].j - jh;
                if (adj > assoc_dj) continue;
                const uint64_t key = assign_key(cands[c].votes, adj, c);
                if (best_c < 0 || key > best) { best = key; best_c = (int32_t)c; }
            }
            hit_to_cand[h] = best_c;
        }
    }
    if (apply_dedup) {
        if (!cand_nhits || !cand_keep) return -1;
        long long n_cands = cand_offsets[n_events] < capacity ? cand_offsets[n_events] : capacity;
        dedup(n_hits, n_cands, min_hits, hit_to_cand, cand_nhits, cand_keep);
    }
    return 0;
}

// D8/D9 -- independent indexed version: a dense per-event volume mapping bin -> candidate index,
// then every hit re-traces ALL its columns (full scan) and probes j in [jh-dj, jh+dj].
int orc_assign_indexed(const orc_binning* b, float bz, const float* hits_xy, int32_t n_hits,
                       const int32_t* event_offsets, int32_t n_events, const orc_candidate* cands,
                       const int32_t* cand_offsets, long long capacity, int32_t assoc_dj, int32_t min_hits,
                       int32_t apply_dedup, int32_t* hit_to_cand, int32_t* cand_nhits, uint8_t* cand_keep) {
    if (!valid_binning(b) || !event_offsets || !cand_offsets || !hit_to_cand) return -1;
    const Tables t = make_tables(*b, bz);
    const int nphi = b->n_phi, nq = b->n_qpt, nd = b->n_d0;
    std::vector<int32_t> index((size_t)nd * nphi * nq, -1);
    for (int e = 0; e < n_events; ++e) {
        long long c0 = cand_offsets[e], c1 = cand_offsets[e + 1];
        if (c1 > capacity) c1 = capacity;
        for (long long c = c0; c < c1; ++c)
            index[((size_t)cands[c].k * nphi + cands[c].i) * nq + cands[c].j] = (int32_t)c;
        for (int h = event_offsets[e]; h < event_offsets[e + 1]; ++h) {
            const float x = hits_xy[2 * (size_t)h], y = hits_xy[2 * (size_t)h + 1];
            const float r2 = hit_r2(x, y);
            uint64_t best = 0;
            int32_t best_c = -1;
            for (int i = 0; i < nphi; ++i)
                for (int k = 0; k < nd; ++k) {
                    const int jh = vote_bin(t, nq, x, y, r2, i, k);
                    if (jh < 0) continue;
                    for (int j = jh - assoc_dj; j <= jh + assoc_dj; ++j) {
                        if (j < 0 || j >= nq) continue;
                        const int32_t c = index[((size_t)k * nphi + i) * nq + j];
                        if (c < 0) continue;
                        const int adj = jh > j ? jh - j : j - jh;
                        const uint64_t key = assign_key(cands[c].votes, adj, c);
                        if (best_c < 0 || key > best) { best = key; best_c = c; }
                    }
                }
            hit_to_cand[h] = best_c;
        }
        for (long long c = c0; c < c1; ++c)
            index[((size_t)cands[c].k * nphi + cands[c].i) * nq + cands[c].j] = -1;
    }
    if (apply_dedup) {
        if (!cand_nhits || !cand_keep) return -1;
        long long n_cands = cand_offsets[n_events] < capacity ? cand_offsets[n_events] : capacity;
        dedup(n_hits, n_cands, min_hits, hit_to_cand, cand_nhits, cand_keep);
    }
    return 0;
}

// D12 -- re-assignment rounds ("all track candidates found ... are cleaned to select only the best candidate
// ... and eliminate duplicate tracks"; "hits in these tracks are then removed, allowing later iterations";
// SURVEY 8(f) f4).  D9 drops a candidate with fewer than min_hits hits and leaves its hits unassigned; here those hits
// re-enter the association.  Round t = 1, 2, ...: every hit takes its best candidate (D8 key) among the candidates
// ALIVE in this round (round 1: all of them); a candidate stays alive iff at least min_hits hits took it.  Stop when no
// candidate was dropped in a round, or after max_rounds rounds.  Outputs: hit_to_cand = the last round's assignment, with
// hits on a candidate dropped in that last round set to -1; cand_keep = alive after the last round; cand_nhits[c] = the
// number of hits c had in the last round in which it was alive (so max_rounds = 1 is exactly D8 + D9).
// Brute force over (hit, candidate) pairs, written out from the definition.  Returns the number of rounds run, < 0 on
// bad arguments.
int orc_assign_rounds(const orc_binning* b, float bz, const float* hits_xy, int32_t n_hits,
                      const int32_t* event_offsets, int32_t n_events, const orc_candidate* cands,
                      const int32_t* cand_offsets, long long capacity, int32_t assoc_dj, int32_t min_hits,
                      int32_t max_rounds, int32_t* hit_to_cand, int32_t* cand_nhits, uint8_t* cand_keep) {
    if (!valid_binning(b) || !event_offsets || !cand_offsets || !hit_to_cand || !cand_nhits || !cand_keep) return -1;
    if (max_rounds < 1) return -1;
    const Tables t = make_tables(*b, bz);
    const long long n_cands = cand_offsets[n_events] < capacity ? cand_offsets[n_events] : capacity;
    std::vector<uint8_t> alive((size_t)(n_cands > 0 ? n_cands : 1), 1);
    std::vector<int32_t> count((size_t)(n_cands > 0 ? n_cands : 1), 0);
    for (long long c = 0; c < n_cands; ++c) cand_nhits[c] = 0;
    int rounds = 0;
    for (;;) {
        ++rounds;
        for (int e = 0; e < n_events; ++e) {
            long long c0 = cand_offsets[e], c1 = cand_offsets[e + 1];
            if (c1 > capacity) c1 = capacity;
            for (int h = event_offsets[e]; h < event_offsets[e + 1]; ++h) {
                const float x = hits_xy[2 * (size_t)h], y = hits_xy[2 * (size_t)h + 1];
                const float r2 = hit_r2(x, y);
                uint64_t best = 0;
                int32_t best_c = -1;
                for (long long c = c0; c < c1; ++c) {
                    if (!alive[(size_t)c]) continue;
                    const int jh = vote_bin(t, b->n_qpt, x, y, r2, cands[c].i, cands[c].k);
                    if (jh < 0) continue;
                    const int adj = jh > cands[c].j ? jh - cands[c].j : cands[c].j - jh;
                    if (adj > assoc_dj) continue;
                    const uint64_t key = assign_key(cands[c].votes, adj, c);
                    if (best_c < 0 || key > best) { best = key; best_c = (int32_t)c; }
                }
                hit_to_cand[h] = best_c;
            }
        }
        for (long long c = 0; c < n_cands; ++c) count[(size_t)c] = 0;
        for (int h = 0; h < n_hits; ++h)
            if (hit_to_cand[h] >= 0) count[(size_t)hit_to_cand[h]] += 1;
        bool dropped = false;
        for (long long c = 0; c < n_cands; ++c) {
            if (!alive[(size_t)c]) continue;
            cand_nhits[c] = count[(size_t)c];
            if (count[(size_t)c] < min_hits) { alive[(size_t)c] = 0; dropped = true; }
        }
        if (!dropped || rounds >= max_rounds) break;
    }
    for (long long c = 0; c < n_cands; ++c) cand_keep[c] = alive[(size_t)c];
    for (int h = 0; h < n_hits; ++h)
        if (hit_to_cand[h] >= 0 && !alive[(size_t)hit_to_cand[h]]) hit_to_cand[h] = -1;
    return rounds;
}

// D10 -- second Hough transform: displaced vertices from the found straight tracks ("apply a Hough
// transform to the track maxima"; Fig. 3: the tracks of one vertex lie on a sinusoid in (phi0, d0)).  A vertex at polar
// position (R, Phi) is on the line (phi0, d0) iff d0 = R sin(Phi - phi0).  Every kept candidate (column i, d0 bin j) of a
// LINE-model track space votes, for every vertex-azimuth column m (the SAME n_phi column centres as the track space), for
// the one compatible radius -- each fp32 operation individually rounded, in this order:
//     tj = (float)j + 0.5f;  dd = tj * wq;  d = qmin + dd;              // centre of the candidate's d0 bin
//     skip the candidate unless keep[c] != 0 and |d| >= d_abs_min       // prompt tracks constrain no vertex
//     sd = sin_m * cos_i - cos_m * sin_i                                 // sin(Phi_m - phi0_i): two products, one subtraction
//     R = d / sd;  t = R * inv_wr;  vote iff 0 <= t < n_r;  n = (int)t;  vacc[e][m][n] += 1
// (R < 0, sd == 0, NaN fall out at the range test; of the two representations (Phi, R), (Phi + pi, -R) exactly one votes).
// vacc: int32 [n_events][n_phi][n_r], zeroed here.  Returns the number of votes, < 0 on bad arguments.
long long orc_vertex_vote(const orc_binning* b, float bz, const orc_candidate* cands, const int32_t* cand_offsets,
                          int32_t n_events, long long capacity, const uint8_t* keep, float d_abs_min, int32_t n_r,
                          float r_max, int32_t* vacc) {
    if (!valid_binning(b) || b->model != 1 || !cand_offsets || !vacc || n_events < 0 || n_r <= 0 || !(r_max > 0.0f)) return -1;
    const Tables t = make_tables(*b, bz);
    const int nphi = b->n_phi;
    const float wq = (float)(((double)b->qpt_max - (double)b->qpt_min) / (double)b->n_qpt);
    const float inv_wr = (float)((double)n_r / (double)r_max);
    std::memset(vacc, 0, sizeof(int32_t) * (size_t)n_events * nphi * n_r);
    long long votes = 0;
    for (int e = 0; e < n_events; ++e) {
        const long long c0 = cand_offsets[e] < capacity ? cand_offsets[e] : capacity;
        const long long c1 = cand_offsets[e + 1] < capacity ? cand_offsets[e + 1] : capacity;
        for (long long c = c0; c < c1; ++c) {
            if (keep && !keep[c]) continue;
            const float tj = (float)cands[c].j + 0.5f;
            const float dd = tj * wq;
            const float d = b->qpt_min + dd;
            if (!(std::fabs(d) >= d_abs_min)) continue;
            const float ci = t.cosT[cands[c].i], si = t.sinT[cands[c].i];
            for (int m = 0; m < nphi; ++m) {
                const float a1 = t.sinT[m] * ci;
                const float a2 = t.cosT[m] * si;
                const float sd = a1 - a2;
                const float R = d / sd;
                const float tt = R * inv_wr;
                if (!(tt >= 0.0f && tt < (float)n_r)) continue;
                vacc[((size_t)e * nphi + m) * n_r + (int)tt] += 1;
                ++votes;
            }
        }
    }
    return votes;
}

// D11 -- circle fit of the hits assigned to each kept candidate ("further computations (e.g., a full Kalman
// fit) can be performed to confirm the existence of the track and obtain the best measurement of the track parameters";
// an algebraic circle fit stands in for the Kalman fit).  Kasa fit, everything in double:
// over the hits h with hit_to_cand[h] == c (x, y = the fp32 coordinates widened to double, z = x x + y y) accumulate
//     n, Sx, Sy, Sz, Sxx, Sxy, Syy, Sxz, Syz
// and minimise sum (z + B x + C y + D)^2:   [Sxx Sxy Sx; Sxy Syy Sy; Sx Sy n] (B, C, D)^T = -(Sxz, Syz, Sz)^T   (Cramer's rule).
// Centre (xc, yc) = (-B/2, -C/2), R^2 = xc^2 + yc^2 - D.  ok = (n >= 3, |det| > 1e-9 * Sxx Syy n scale, R^2 > 0, |centre| > 0).
// Track parameters in the D1 convention, orientation taken from the candidate's column (theta_i in double):
//     p0 = centre (1 - R / |centre|)                      point of the circle closest to the origin
//     t  = +-(-yc, xc) / |centre|, the sign with t . (cos theta_i, sin theta_i) >= 0;   phi0 = atan2(t_y, t_x) in [0, 2pi)
//     n = (-t_y, t_x);   d0 = p0 . n;   1/rho = (centre - p0) . n;   q/pT = -rho / (K Bz)   (0 when Bz == 0)
// out: double fit[c][4] = {phi0, qpt, d0, R};  int32 n_fit[c] = hits used, or -n when the fit is not ok (0: no hits / dropped).
int orc_fit_circles(const orc_binning* b, float bz, const float* hits_xy, int32_t n_hits, const int32_t* hit_to_cand,
                    const orc_candidate* cands, long long n_cands, const uint8_t* keep, double* fit, int32_t* n_fit) {
    if (!valid_binning(b) || !hit_to_cand || !fit || !n_fit || n_hits < 0 || n_cands < 0) return -1;
    std::vector<double> m((size_t)n_cands * 9, 0.0);
    for (int h = 0; h < n_hits; ++h) {
        const long long c = hit_to_cand[h];
        if (c < 0 || c >= n_cands) continue;
        const double x = (double)hits_xy[2 * h], y = (double)hits_xy[2 * h + 1];
        const double z = x * x + y * y;
        double* a = &m[(size_t)c * 9];
        a[0] += 1.0; a[1] += x; a[2] += y; a[3] += z; a[4] += x * x; a[5] += x * y; a[6] += y * y; a[7] += x * z; a[8] += y * z;
    }
    const double kb = kGeVPerTeslaCm * (double)bz;
    for (long long c = 0; c < n_cands; ++c) {
        double* f = fit + 4 * c;
        f[0] = f[1] = f[2] = f[3] = 0.0;
        n_fit[c] = 0;
        if (keep && !keep[c]) continue;
        const double* a = &m[(size_t)c * 9];
        const double n = a[0], Sx = a[1], Sy = a[2], Sz = a[3], Sxx = a[4], Sxy = a[5], Syy = a[6], Sxz = a[7], Syz = a[8];
        const int ni = (int)n;
        if (ni == 0) continue;
        n_fit[c] = -ni;
        if (ni < 3) continue;
        const double det = Sxx * (Syy * n - Sy * Sy) - Sxy * (Sxy * n - Sy * Sx) + Sx * (Sxy * Sy - Syy * Sx);
        if (!(std::fabs(det) > 1.0e-9 * std::fabs(Sxx * Syy * n))) continue;
        const double r1 = -Sxz, r2 = -Syz, r3 = -Sz;
        const double B = (r1 * (Syy * n - Sy * Sy) - Sxy * (r2 * n - Sy * r3) + Sx * (r2 * Sy - Syy * r3)) / det;
        const double Cc = (Sxx * (r2 * n - r3 * Sy) - r1 * (Sxy * n - Sy * Sx) + Sx * (Sxy * r3 - r2 * Sx)) / det;
        const double D = (Sxx * (Syy * r3 - Sy * r2) - Sxy * (Sxy * r3 - r2 * Sx) + r1 * (Sxy * Sy - Syy * Sx)) / det;
        const double xc = -0.5 * B, yc = -0.5 * Cc;
        const double R2 = xc * xc + yc * yc - D;
        const double cn = std::sqrt(xc * xc + yc * yc);
        if (!(R2 > 0.0) || !(cn > 0.0)) continue;
        const double R = std::sqrt(R2);
        const double theta = ((double)cands[c].i + 0.5) * (2.0 * kPi / (double)b->n_phi);
        double tx = -yc / cn, ty = xc / cn;
        if (tx * std::cos(theta) + ty * std::sin(theta) < 0.0) { tx = -tx; ty = -ty; }
        const double s = 1.0 - R / cn;
        const double p0x = xc * s, p0y = yc * s;
        const double nx = -ty, ny = tx;
        double phi0 = std::atan2(ty, tx);
        if (phi0 < 0.0) phi0 += 2.0 * kPi;
        const double inv_rho = (xc - p0x) * nx + (yc - p0y) * ny;
        f[0] = phi0;
        f[1] = (kb != 0.0) ? -(1.0 / inv_rho) / kb : 0.0;
        f[2] = p0x * nx + p0y * ny;
        f[3] = R;
        n_fit[c] = ni;
    }
    return 0;
}

}  // extern "C"

// windows.cu -- host-only: radius classes and conservative phi0-column windows (work sizing for A1/A2/A5).
//
// For a hit at radius r and azimuth phi, and a d0 slice with centre d0, the D3 test
//     qmin <= v < qmax,   v = (d0 - r s) / (A (r^2 - 2 d0 r s + d0^2)),   s = sin(phi - phi0),   f = r cos(phi - phi0) > 0
// is, for A > 0 and c(q) = 1 - 2 q A d0 > 0, the pair of LINEAR inequalities in s
//     S(qmax) < s <= S(qmin),      S(q) = (d0 - q A (r^2 + d0^2)) / (r c(q)) = a(q)/r - b(q) r,
// so the columns a hit votes in are one contiguous cyclic run  phi0 - phi in [-asin(S(qmin)), -asin(S(qmax))]
// (DESIGN.md "Windows").  The kernels evaluate the exact fp32 D3 sequence at every column of a window that
// CONTAINS that run, so a window changes how much work is done, never a result (include/hough.h, S19).
//
// Hits are grouped into radius classes (narrow ones around the detector layers, wide ones elsewhere, an
// open-ended last one); the table holds, per (class, d0 slice), the hull of the run over the class's radius
// interval as  lo_off  (columns, relative to the hit's column coordinate u = phi/dphi - 0.5) and the number
// of columns `steps` to visit starting at ceil(u + lo_off).
#include <algorithm>
#include <cmath>
#include <vector>

#include "common.cuh"

namespace {

const double kPi = 3.14159265358979323846;

// hull of S(q; r) = a/r - b r over r in [ra, rb]  (ra may be 0)
void hull_S(double a, double b, double ra, double rb, double& smin, double& smax) {
    auto S = [&](double r) {
        if (r <= 0.0) return a > 0 ? 1e30 : (a < 0 ? -1e30 : 0.0);
        return a / r - b * r;
    };
    smin = std::min(S(ra), S(rb));
    smax = std::max(S(ra), S(rb));
    if (b != 0.0 && -a / b > 0.0) {                 // interior extremum at r* = sqrt(-a/b)
        const double rs = std::sqrt(-a / b);
        if (rs > ra && rs < rb) { smin = std::min(smin, S(rs)); smax = std::max(smax, S(rs)); }
    }
}

}  // namespace

int hough_build_windows(const hough_binning& b, float bz, int n_layers, const float* layer_r, HoughWindows& out) {
    const int nphi = b.n_phi, nd = b.n_d0;
    const double A = (double)(float)(0.5 * 0.00299792458 * (double)bz);
    const double qmin = b.qpt_min, qmax = b.qpt_max;
    const double qabs = std::max(std::fabs(qmin), std::fabs(qmax));

    // ---- radius classes -------------------------------------------------------------------------------
    std::vector<double> R;
    for (int l = 0; l < n_layers; ++l)
        if (std::isfinite(layer_r[l]) && layer_r[l] > 0.0f) R.push_back((double)layer_r[l]);
    std::sort(R.begin(), R.end());
    double r_top;
    if (!R.empty()) r_top = 1.25 * R.back();
    else r_top = (A > 0 && qabs > 0) ? std::min(1.0 / (A * qabs), 1.0e3) : 100.0;
    const double tau = 2.0e-4;                       // narrow class half-width (relative) around a layer
    std::vector<double> edges;
    for (int wide = 48; ; wide = wide * 3 / 4) {
        edges.assign(1, 0.0);
        const double wmax = r_top / (double)wide;
        auto fill_to = [&](double hi) {
            const double cur = edges.back();
            if (hi <= cur) return;
            const int n = std::max(1, (int)std::ceil((hi - cur) / wmax));
            for (int t = 1; t <= n; ++t) edges.push_back(cur + (hi - cur) * (double)t / (double)n);
        };
        for (double r : R) {
            fill_to(r * (1.0 - tau));
            if (r * (1.0 + tau) > edges.back()) edges.push_back(r * (1.0 + tau));
        }
        fill_to(r_top);
        if ((int)edges.size() <= HOUGH_MAX_CLASSES || wide <= 2) break;     // edges.size() = classes incl. open one
    }
    if ((int)edges.size() > HOUGH_MAX_CLASSES) edges.resize(HOUGH_MAX_CLASSES);
    const int nc = (int)edges.size();                // classes 0..nc-2 bounded, class nc-1 = [edges[nc-1], inf)
    out.n_class = nc;
    out.edge2.resize(nc);
    for (int c = 0; c < nc; ++c) out.edge2[c] = (float)(edges[c] * edges[c]);
    out.edge2[0] = 0.0f;
    out.lo_off.assign((size_t)nc * nd, 0.0f);
    out.steps.assign((size_t)nc * nd, 0);
    out.fwd_safe.assign((size_t)nc * nd, 0);

    // ---- windows --------------------------------------------------------------------------------------
    const double dphi = 2.0 * kPi / (double)nphi;
    const double margin_cols = 0.25 + 2.0e-6 * (double)nphi;
    const double eps_q = 1.0e-5 * (std::fabs(qmin) + std::fabs(qmax));
    const float full_lo = (float)(-(double)(nphi / 4) - 2.0);
    const int full_steps = std::min(nphi, nphi / 2 + 5);
    for (int c = 0; c < nc; ++c) {
        const bool open = c == nc - 1;
        const double ra = std::sqrt((double)out.edge2[c]) * (1.0 - 1.0e-6);
        const double rb = open ? 0.0 : std::sqrt((double)(float)(edges[c + 1] * edges[c + 1])) * (1.0 + 1.0e-6);
        for (int k = 0; k < nd; ++k) {
            float& lo = out.lo_off[(size_t)c * nd + k];
            int& st = out.steps[(size_t)c * nd + k];
            lo = full_lo; st = full_steps;           // default: the whole forward half (always contains the run)
            if (open) continue;
            if (b.model == HOUGH_MODEL_LINE) {
                // D3L: qmin <= r s < qmax (cm), s = sin(phi - phi0): s in [qmin / r, qmax / r) over the class's radii
                if (!(ra > 0.0)) continue;
                const double eps_d = 1.0e-5 * (std::fabs(qmin) + std::fabs(qmax));
                double s_lo = std::min((qmin - eps_d) / ra, (qmin - eps_d) / rb);
                double s_hi = std::max((qmax + eps_d) / ra, (qmax + eps_d) / rb);
                s_lo -= 1.0e-5 + 1.0e-6 * std::fabs(s_lo);
                s_hi += 1.0e-5 + 1.0e-6 * std::fabs(s_hi);
                if (s_lo > 1.0 || s_hi < -1.0 || s_lo > s_hi) { lo = 0.0f; st = 0; continue; }
                const double d_lo = -std::asin(std::min(s_hi, 1.0));
                const double d_hi = -std::asin(std::max(s_lo, -1.0));
                const double lo_c = d_lo / dphi - margin_cols, hi_c = d_hi / dphi + margin_cols;
                const int steps = (int)std::floor(hi_c - lo_c) + 1;
                if (steps >= full_steps) continue;
                lo = (float)lo_c;
                if ((double)lo > lo_c) lo = std::nextafterf(lo, -1.0e30f);
                st = steps + 1;
                const double lim = 89.0 / 360.0 * (double)nphi;
                if (c > 0 && (double)lo - 2.0 >= -lim && (double)lo + (double)st + 3.0 <= lim)
                    out.fwd_safe[(size_t)c * nd + k] = 1;
                continue;
            }
            if (!(A > 0.0)) continue;
            double d0 = 0.0;
            if (nd > 1)
                d0 = (double)(float)((double)b.d0_min + ((double)k + 0.5) * ((double)b.d0_max - (double)b.d0_min) / (double)nd);
            const double qlo = qmin - eps_q, qhi = qmax + eps_q;
            const double c_lo = 1.0 - 2.0 * qlo * A * d0, c_hi = 1.0 - 2.0 * qhi * A * d0;
            if (!(c_lo > 1.0e-3) || !(c_hi > 1.0e-3)) continue;
            // s <= S(qlo) and s > S(qhi)
            double t0, t1, s_hi, s_lo;
            hull_S(d0 * (1.0 - qlo * A * d0) / c_lo, qlo * A / c_lo, ra, rb, t0, s_hi);
            hull_S(d0 * (1.0 - qhi * A * d0) / c_hi, qhi * A / c_hi, ra, rb, s_lo, t1);
            (void)t0; (void)t1;
            if (!std::isfinite(s_lo) || !std::isfinite(s_hi)) continue;
            s_lo -= 1.0e-5 + 1.0e-6 * std::fabs(s_lo);
            s_hi += 1.0e-5 + 1.0e-6 * std::fabs(s_hi);
            if (s_lo > 1.0 || s_hi < -1.0 || s_lo > s_hi) { lo = 0.0f; st = 0; continue; }   // no column can pass
            const double d_lo = -std::asin(std::min(s_hi, 1.0));      // phi0 - phi, radians
            const double d_hi = -std::asin(std::max(s_lo, -1.0));
            const double lo_c = d_lo / dphi - margin_cols, hi_c = d_hi / dphi + margin_cols;
            const int steps = (int)std::floor(hi_c - lo_c) + 1;
            if (steps >= full_steps) continue;
            lo = (float)lo_c;
            if ((double)lo > lo_c) lo = std::nextafterf(lo, -1.0e30f);
            st = steps + 1;                           // +1: the float rounding of u + lo_off on the device
            // Every column of the window, one before it and two after it (the walk visits even/odd column pairs) is
            // within 89 degrees of the hit's azimuth and the class excludes r = 0:
            // f = r cos(phi0 - phi) >= 0.017 r exceeds its fp32 rounding error (2^-23 r) by far, so the D3 forward
            // test passes at every column of the window and the walk's fast path may skip it.
            const double lim = 89.0 / 360.0 * (double)nphi;
            if (c > 0 && ra > 0.0 && (double)lo - 2.0 >= -lim && (double)lo + (double)st + 3.0 <= lim)
                out.fwd_safe[(size_t)c * nd + k] = 1;
        }
    }
    return HOUGH_OK;
}

extern "C" int hough_window_table(const hough_binning* b, const hough_geometry* g, int32_t* n_class, float* edge_r2,
                                  float* lo_off, int32_t* steps) {
    if (!b || !g || !n_class) return HOUGH_ERR_INVALID_ARG;
    if (b->n_phi <= 0 || b->n_phi % 4 != 0 || b->n_qpt <= 0 || b->n_d0 <= 0) return HOUGH_ERR_INVALID_ARG;
    if (g->n_layers < 0 || g->n_layers > 64 || (g->n_layers > 0 && !g->layer_radius_cm)) return HOUGH_ERR_INVALID_ARG;
    HoughWindows w;
    const int rc = hough_build_windows(*b, g->bz_tesla, g->n_layers, g->layer_radius_cm, w);
    if (rc != HOUGH_OK) return rc;
    *n_class = w.n_class;
    if (edge_r2) std::copy(w.edge2.begin(), w.edge2.end(), edge_r2);
    if (lo_off) std::copy(w.lo_off.begin(), w.lo_off.end(), lo_off);
    if (steps) std::copy(w.steps.begin(), w.steps.end(), steps);
    return HOUGH_OK;
}

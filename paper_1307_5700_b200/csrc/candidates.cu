// Host candidate stage (BASELINE.json north_star: "DBSCAN-style clustering and the analytic DM-SNR
// candidate filter stay on the host"): FDBSCAN over the (time, DM, SNR) detections and the eight-step
// DM-SNR-curve classifier with Eqs. 3 and 4.  Plain host C++ (no device work); region queries go
// through a uniform grid of eps-sized cells instead of the O(N^2) scan of the oracle.
#include <algorithm>
#include <cmath>
#include <unordered_map>
#include <vector>

#include "mdsm_internal.h"

namespace {

struct Point { double x[3]; };

struct Grid {
    const std::vector<Point> &pts;
    double eps[3];
    std::unordered_map<uint64_t, std::vector<int32_t>> cells;

    static uint64_t key(int64_t a, int64_t b, int64_t c)
    {
        // 21 bits per coordinate after an offset: collisions only merge candidate lists, the box test decides
        return ((uint64_t)(a + (1 << 20)) & 0x1fffff) << 42 | ((uint64_t)(b + (1 << 20)) & 0x1fffff) << 21 | ((uint64_t)(c + (1 << 20)) & 0x1fffff);
    }
    int64_t cell(int dim, double v) const { return (int64_t)std::floor(v / eps[dim]); }

    Grid(const std::vector<Point> &p, const double *e) : pts(p)
    {
        for (int k = 0; k < 3; ++k) eps[k] = e[k];
        cells.reserve(p.size());
        for (size_t i = 0; i < p.size(); ++i)
            cells[key(cell(0, p[i].x[0]), cell(1, p[i].x[1]), cell(2, p[i].x[2]))].push_back((int32_t)i);
    }

    // every point q with |x_q[k] - x_p[k]| <= eps[k] in all three dimensions, ascending index order (p itself included)
    void query(int32_t p, std::vector<int32_t> &out) const
    {
        out.clear();
        const Point &c = pts[p];
        const int64_t c0 = cell(0, c.x[0]), c1 = cell(1, c.x[1]), c2 = cell(2, c.x[2]);
        for (int64_t a = c0 - 1; a <= c0 + 1; ++a)
            for (int64_t b = c1 - 1; b <= c1 + 1; ++b)
                for (int64_t d = c2 - 1; d <= c2 + 1; ++d) {
                    auto it = cells.find(key(a, b, d));
                    if (it == cells.end()) continue;
                    for (int32_t q : it->second) {
                        const Point &o = pts[q];
                        if (std::fabs(o.x[0] - c.x[0]) <= eps[0] && std::fabs(o.x[1] - c.x[1]) <= eps[1] && std::fabs(o.x[2] - c.x[2]) <= eps[2])
                            out.push_back(q);
                    }
                }
        std::sort(out.begin(), out.end());
        out.erase(std::unique(out.begin(), out.end()), out.end());     // a key collision can list a cell twice
    }
};

constexpr int32_t kUnclassified = -2, kNoise = -1;

// One beam's detections, points in the caller's order.  exact = 1: DBSCAN (every neighbour of a core point is expanded);
// exact = 0: FDBSCAN: only the representative border points of a core point's neighbourhood -- per
// dimension and direction the neighbour of this cluster farthest from the core point, the lowest index among equals --
// are expanded, each point at most once.
int64_t cluster_beam(const std::vector<Point> &pts, const double *eps, int min_pts, bool exact, int32_t *label, int32_t first_id,
                     int64_t *n_queries)
{
    const int32_t n = (int32_t)pts.size();
    Grid grid(pts, eps);
    std::vector<int32_t> nb, queue;
    std::vector<uint8_t> done(n, 0);            // DBSCAN: queued; FDBSCAN: expanded
    for (int32_t i = 0; i < n; ++i) label[i] = kUnclassified;
    int32_t cid = first_id;
    for (int32_t p = 0; p < n; ++p) {
        if (label[p] != kUnclassified) continue;
        grid.query(p, nb);
        ++*n_queries;
        if ((int)nb.size() < min_pts) { label[p] = kNoise; continue; }
        queue.clear();
        size_t head = 0;
        if (exact) {
            label[p] = cid;
            queue.push_back(p);
            done[p] = 1;
            while (head < queue.size()) {
                const int32_t q = queue[head++];
                grid.query(q, nb);
                ++*n_queries;
                if ((int)nb.size() < min_pts) continue;
                for (int32_t r : nb) {
                    if (label[r] == kUnclassified || label[r] == kNoise) label[r] = cid;
                    if (label[r] == cid && !done[r]) { queue.push_back(r); done[r] = 1; }
                }
            }
        } else {
            queue.push_back(p);
            bool first = true;
            while (head < queue.size()) {
                const int32_t q = queue[head++];
                if (done[q]) continue;
                done[q] = 1;
                if (!first) { grid.query(q, nb); ++*n_queries; }
                first = false;
                if ((int)nb.size() < min_pts) continue;
                for (int32_t r : nb)
                    if (label[r] == kUnclassified || label[r] == kNoise) label[r] = cid;
                for (int dim = 0; dim < 3; ++dim)
                    for (int dir = 1; dir >= -1; dir -= 2) {
                        int32_t best = -1;
                        double bestv = 0.0;
                        for (int32_t r : nb) {
                            if (label[r] != cid) continue;
                            const double v = (double)dir * (pts[r].x[dim] - pts[q].x[dim]);
                            if (v > bestv) { bestv = v; best = r; }
                        }
                        if (best >= 0 && !done[best]) queue.push_back(best);
                    }
            }
        }
        ++cid;
    }
    return cid - first_id;
}

// Eq. 3 with Eq. 4
double dm_curve(double ddm, double bw_mhz, double w_ms, double nu_ghz)
{
    const double zeta = std::fabs(6.91e-3 * ddm * bw_mhz / (w_ms * (nu_ghz * nu_ghz * nu_ghz)));
    if (zeta < 1e-12) return 1.0;
    return 0.5 * std::sqrt(3.14159265358979323846) * std::erf(zeta) / zeta;
}

}  // namespace

extern "C" int mdsm_cluster_events(const mdsm_event *h_events, int64_t n, double dm_low, double dm_step, double eps_t,
                                   double eps_dm, double eps_snr, int min_pts, int exact, int32_t *h_labels,
                                   int64_t *h_nclusters, int64_t *h_nqueries)
{
    MDSM_REQUIRE(n >= 0 && (n == 0 || (h_events && h_labels)) && h_nclusters, "null argument");
    MDSM_REQUIRE(eps_t > 0.0 && eps_dm > 0.0 && eps_snr > 0.0 && min_pts >= 1, "eps_t, eps_dm, eps_snr must be > 0 and min_pts >= 1");
    MDSM_REQUIRE(n < ((int64_t)1 << 31), "at most 2^31 - 1 events");
    const double eps[3] = {eps_t, eps_dm, eps_snr};
    // beams are clustered one by one (a detection list per beam), in order of first appearance
    std::vector<int32_t> beams;
    std::unordered_map<int32_t, std::vector<int64_t>> by_beam;
    for (int64_t i = 0; i < n; ++i) {
        auto it = by_beam.find(h_events[i].beam);
        if (it == by_beam.end()) { beams.push_back(h_events[i].beam); it = by_beam.emplace(h_events[i].beam, std::vector<int64_t>()).first; }
        it->second.push_back(i);
    }
    int64_t ncl = 0, nq = 0;
    std::vector<Point> pts;
    std::vector<int32_t> lab;
    for (int32_t b : beams) {
        const std::vector<int64_t> &idx = by_beam[b];
        pts.resize(idx.size());
        lab.resize(idx.size());
        for (size_t k = 0; k < idx.size(); ++k) {
            const mdsm_event &e = h_events[idx[k]];
            pts[k].x[0] = (double)e.t;
            pts[k].x[1] = dm_low + (double)e.dm_idx * dm_step;
            pts[k].x[2] = (double)e.snr;
        }
        ncl += cluster_beam(pts, eps, min_pts, exact != 0, lab.data(), (int32_t)ncl, &nq);
        for (size_t k = 0; k < idx.size(); ++k) h_labels[idx[k]] = lab[k];
    }
    *h_nclusters = ncl;
    if (h_nqueries) *h_nqueries = nq;
    return MDSM_OK;
}

extern "C" int mdsm_classify_clusters(const mdsm_event *h_events, const int32_t *h_labels, int64_t n, int64_t nclusters,
                                      double dm_low, double dm_step, double tsamp, double bw_mhz, double nu_ghz, int k_smooth,
                                      double rmse_max, double *h_results)
{
    MDSM_REQUIRE(n >= 0 && nclusters >= 0 && (n == 0 || (h_events && h_labels)) && (nclusters == 0 || h_results), "null argument");
    MDSM_REQUIRE(k_smooth >= 1 && (k_smooth & 1) && tsamp > 0.0 && bw_mhz > 0.0 && nu_ghz > 0.0, "k_smooth must be odd, tsamp, bandwidth and frequency > 0");
    std::vector<std::vector<int64_t>> members((size_t)nclusters);
    for (int64_t i = 0; i < n; ++i) {
        MDSM_REQUIRE(h_labels[i] < nclusters, "label %d out of range", h_labels[i]);
        if (h_labels[i] >= 0) members[(size_t)h_labels[i]].push_back(i);
    }
    std::vector<double> sig, sm;
    std::vector<int64_t> cnt;
    for (int64_t c = 0; c < nclusters; ++c) {
        double *res = h_results + 5 * c;
        const std::vector<int64_t> &m = members[(size_t)c];
        if (m.empty()) { res[0] = -1.0; res[1] = res[2] = res[3] = res[4] = 0.0; continue; }
        int dmin = h_events[m[0]].dm_idx, dmax = dmin;
        for (int64_t i : m) { dmin = std::min(dmin, h_events[i].dm_idx); dmax = std::max(dmax, h_events[i].dm_idx); }
        const int nd = dmax - dmin + 1;
        sig.assign(nd, 0.0); sm.assign(nd, 0.0); cnt.assign(nd, 0);
        for (int64_t i : m) {                                              // 1: collapse the time dimension
            const int d = h_events[i].dm_idx - dmin;
            if (cnt[d] == 0 || (double)h_events[i].snr > sig[d]) sig[d] = (double)h_events[i].snr;
            ++cnt[d];
        }
        const int h = k_smooth / 2;                                        // 2: k-element moving average
        for (int d = 0; d < nd; ++d) {
            double s = 0.0; int k = 0;
            for (int e = std::max(0, d - h); e <= std::min(nd - 1, d + h); ++e) { s += sig[e]; ++k; }
            sm[d] = s / (double)k;
        }
        int dstar = 0;                                                     // 3: the DM with the most detections
        for (int d = 1; d < nd; ++d) if (cnt[d] > cnt[dstar]) dstar = d;
        const double dm_star = dm_low + (double)(dstar + dmin) * dm_step;
        int32_t t0 = 0, t1 = 0; bool have = false;                         // 4: width at that DM
        for (int64_t i : m)
            if (h_events[i].dm_idx - dmin == dstar) {
                if (!have || h_events[i].t < t0) t0 = h_events[i].t;
                if (!have || h_events[i].t > t1) t1 = h_events[i].t;
                have = true;
            }
        const double w_ms = (double)(t1 - t0 + 1) * tsamp * 1e3;
        res[1] = (double)(dstar + dmin); res[2] = sig[dstar]; res[3] = w_ms;
        if (dm_star < 1.0) { res[0] = 1.0; res[4] = 0.0; continue; }       //    DM < 1: broadband RFI
        double mx = 0.0;                                                   // 5: normalise
        for (int d = 0; d < nd; ++d) mx = std::max(mx, sm[d]);
        double se = 0.0;                                                   // 6, 7: model curve and RMSE
        for (int d = 0; d < nd; ++d) {
            const double ddm = (dm_low + (double)(d + dmin) * dm_step) - dm_star;
            const double e = dm_curve(ddm, bw_mhz, w_ms, nu_ghz) - (mx > 0.0 ? sm[d] / mx : 0.0);
            se += e * e;
        }
        res[4] = std::sqrt(se / (double)nd);
        res[0] = res[4] > rmse_max ? 2.0 : 0.0;                            // 8
    }
    return MDSM_OK;
}

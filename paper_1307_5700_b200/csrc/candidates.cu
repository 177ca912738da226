// Host candidate stage (BASELINE.json north_star: "DBSCAN-style clustering and the analytic DM-SNR
// candidate filter stay on the host"): FDBSCAN over the (time, DM, SNR) detections and the eight-step
// DM-SNR-curve classifier with Eqs. 3 and 4.  Plain host C++ (no device work).  Region queries go
// through a uniform grid of eps-sized cells; the six FDBSCAN representatives come out of one sweep over a neighbour
// list; the classifier works on a DM-sorted event list reduced to one row per DM trial.
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

// ---- density clustering of one beam's detections ------------------------------------------------------------------
// PAPER.md:118-126.  A cluster is grown from a core point ("seed") through a FIFO of points still to be examined.
// DBSCAN (exact): every member found goes through the FIFO.  FDBSCAN: of a core point's neighbourhood only
// the six border representatives do -- "two for each dimension, one for each direction when placing the core point at
// the origin" -- found in ONE sweep over the neighbour list that keeps, per (dimension, direction) slot, the member of the
// growing cluster with the largest displacement (strictly positive; neighbour lists are ascending, so the first of
// equally far points stays).  Neighbour lists come from the grid above.
class BeamClusterer {
public:
    BeamClusterer(const std::vector<Point> &pts, const double *eps, int min_pts, int32_t *label)
        : pts_(pts), grid_(pts, eps), min_pts_(min_pts), label_(label), in_fifo_(pts.size(), 0)
    {
        std::fill(label_, label_ + pts.size(), kFresh);
    }

    // Returns the number of clusters found; ids start at first_id.
    int64_t run(bool exact, int32_t first_id)
    {
        int32_t next_id = first_id;
        for (int32_t p = 0; p < (int32_t)pts_.size(); ++p) {
            if (label_[p] != kFresh) continue;
            if (!core_neighbourhood(p)) { label_[p] = kNoiseLabel; continue; }
            cid_ = next_id++;
            fifo_.clear();
            in_fifo_[p] = 1;                                   // the seed is being examined right now, with nb_ in hand
            absorb(exact);
            for (size_t head = 0; head < fifo_.size(); ++head)
                if (core_neighbourhood(fifo_[head])) { centre_ = fifo_[head]; absorb(exact); }
        }
        return next_id - first_id;
    }
    int64_t queries() const { return queries_; }

private:
    static constexpr int32_t kFresh = -2, kNoiseLabel = -1;

    // Region query around p into nb_; true when p is a core point.  Sets centre_.
    bool core_neighbourhood(int32_t p)
    {
        centre_ = p;
        grid_.query(p, nb_);
        ++queries_;
        return (int)nb_.size() >= min_pts_;
    }

    void enqueue(int32_t r)
    {
        if (in_fifo_[r]) return;                               // examined, or waiting to be: a point is examined once
        in_fifo_[r] = 1;
        fifo_.push_back(r);
    }

    // nb_ is the neighbourhood of the core point centre_: its unclaimed points (fresh or noise) join the cluster, then the
    // points to examine next are queued: all members (DBSCAN) or the six representatives (FDBSCAN).
    void absorb(bool exact)
    {
        int32_t far[6] = {-1, -1, -1, -1, -1, -1};             // slot 2 * dim + (0: towards larger, 1: towards smaller values)
        double reach[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        const Point &c = pts_[centre_];
        for (int32_t r : nb_) {
            if (label_[r] < 0) label_[r] = cid_;
            if (label_[r] != cid_) continue;                   // a border point another cluster claimed first stays there
            if (exact) { enqueue(r); continue; }
            for (int dim = 0; dim < 3; ++dim) {
                const double off = pts_[r].x[dim] - c.x[dim];
                const int slot = 2 * dim + (off < 0.0 ? 1 : 0);
                if (std::fabs(off) > reach[slot]) { reach[slot] = std::fabs(off); far[slot] = r; }
            }
        }
        if (!exact)
            for (int slot = 0; slot < 6; ++slot)
                if (far[slot] >= 0) enqueue(far[slot]);
    }

    const std::vector<Point> &pts_;
    Grid grid_;
    int min_pts_;
    int32_t *label_;
    std::vector<uint8_t> in_fifo_;
    std::vector<int32_t> nb_, fifo_;
    int32_t centre_ = 0, cid_ = 0;
    int64_t queries_ = 0;
};

// ---- DM-SNR classifier ---------------------------------------------------------------------------------------------
// Eq. 3 at the zeta of Eq. 4: the fraction of a pulse's peak that survives dedispersion at a
// DM that is ddm off, for a pulse of width w_ms observed over bw_mhz at nu_ghz.
double surviving_fraction(double ddm, double bw_mhz, double w_ms, double nu_ghz)
{
    const double zeta = std::fabs(6.91e-3 * ddm * bw_mhz / (w_ms * (nu_ghz * nu_ghz * nu_ghz)));
    return zeta < 1e-12 ? 1.0 : 0.5 * std::sqrt(3.14159265358979323846) * std::erf(zeta) / zeta;
}

// What the detections of one cluster at one DM trial collapse to (PAPER.md:146 step 1: "collapsing the time dimension").
struct DmRow {
    int32_t dm_idx;
    int64_t count;        // detections at this DM
    double peak;          // the strongest of them
    int32_t t_first, t_last;
};

// Steps 1-8 of PAPER.md:144-156 for one cluster; `order` lists its events sorted by DM index.
void classify_one(const mdsm_event *ev, const int64_t *order, int64_t m, double dm_low, double dm_step, double tsamp, double bw_mhz,
                  double nu_ghz, int k_smooth, double rmse_max, std::vector<DmRow> &rows, std::vector<double> &sig, double *res)
{
    // 1: one sweep over the DM-sorted events gives a row per DM that has detections
    rows.clear();
    for (int64_t k = 0; k < m; ++k) {
        const mdsm_event &e = ev[order[k]];
        if (rows.empty() || rows.back().dm_idx != e.dm_idx) rows.push_back(DmRow{e.dm_idx, 0, (double)e.snr, e.t, e.t});
        DmRow &r = rows.back();
        r.count += 1;
        r.peak = std::max(r.peak, (double)e.snr);
        r.t_first = std::min(r.t_first, e.t);
        r.t_last = std::max(r.t_last, e.t);
    }
    // 3, 4: the DM with the most detections (the lowest such DM), its strongest detection, the pulse width there
    const DmRow *best = &rows[0];
    for (const DmRow &r : rows)
        if (r.count > best->count) best = &r;
    const double dm_best = dm_low + (double)best->dm_idx * dm_step;
    const double w_ms = (double)(best->t_last - best->t_first + 1) * tsamp * 1e3;
    res[1] = (double)best->dm_idx; res[2] = best->peak; res[3] = w_ms;
    if (dm_best < 1.0) { res[0] = 1.0; res[4] = 0.0; return; }           // broadband RFI (step 3)
    // the signature on the dense DM axis of the cluster (0 where a DM trial has no detection)
    const int32_t d_lo = rows.front().dm_idx;
    const int nd = rows.back().dm_idx - d_lo + 1;
    sig.assign((size_t)nd, 0.0);
    for (const DmRow &r : rows) sig[(size_t)(r.dm_idx - d_lo)] = r.peak;
    // 2, 5: centred k-element moving average (shorter at the two ends), then its maximum for the normalisation
    const int half = k_smooth / 2;
    std::vector<double> &smooth = sig;                                      // smoothed values are appended behind the raw ones
    smooth.resize((size_t)2 * nd);
    double top = 0.0;
    for (int d = 0; d < nd; ++d) {
        const int lo = std::max(0, d - half), hi = std::min(nd - 1, d + half);
        double acc = 0.0;
        for (int e = lo; e <= hi; ++e) acc += sig[(size_t)e];
        smooth[(size_t)nd + d] = acc / (double)(hi - lo + 1);
        top = std::max(top, smooth[(size_t)nd + d]);
    }
    // 6, 7: squared distance between the model curve around dm_best and the normalised signature
    double sq = 0.0;
    for (int d = 0; d < nd; ++d) {
        const double ddm = (dm_low + (double)(d + d_lo) * dm_step) - dm_best;
        const double shape = top > 0.0 ? smooth[(size_t)nd + d] / top : 0.0;
        const double miss = surviving_fraction(ddm, bw_mhz, w_ms, nu_ghz) - shape;
        sq += miss * miss;
    }
    res[4] = std::sqrt(sq / (double)nd);
    res[0] = res[4] > rmse_max ? 2.0 : 0.0;                                  // 8
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
        BeamClusterer clusterer(pts, eps, min_pts, lab.data());
        ncl += clusterer.run(exact != 0, (int32_t)ncl);
        nq += clusterer.queries();
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
    // group the events by cluster (counting sort on the label), then order each group by DM index
    std::vector<int64_t> start((size_t)nclusters + 1, 0), order;
    for (int64_t i = 0; i < n; ++i) {
        MDSM_REQUIRE(h_labels[i] < nclusters, "label %d out of range", h_labels[i]);
        if (h_labels[i] >= 0) ++start[(size_t)h_labels[i] + 1];
    }
    for (int64_t c = 0; c < nclusters; ++c) start[(size_t)c + 1] += start[(size_t)c];
    order.resize((size_t)start[(size_t)nclusters]);
    {
        std::vector<int64_t> fill(start.begin(), start.end() - 1);
        for (int64_t i = 0; i < n; ++i)
            if (h_labels[i] >= 0) order[(size_t)fill[(size_t)h_labels[i]]++] = i;
    }
    std::vector<DmRow> rows;
    std::vector<double> sig;
    for (int64_t c = 0; c < nclusters; ++c) {
        double *res = h_results + 5 * c;
        int64_t *first = order.data() + start[(size_t)c];
        const int64_t m = start[(size_t)c + 1] - start[(size_t)c];
        if (m == 0) { res[0] = -1.0; res[1] = res[2] = res[3] = res[4] = 0.0; continue; }
        std::stable_sort(first, first + m, [&](int64_t a, int64_t b) { return h_events[a].dm_idx < h_events[b].dm_idx; });
        classify_one(h_events, first, m, dm_low, dm_step, tsamp, bw_mhz, nu_ghz, k_smooth, rmse_max, rows, sig, res);
    }
    return MDSM_OK;
}

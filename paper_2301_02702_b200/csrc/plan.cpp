// plan.cpp -- host side of the hot path, fp64:
//   a1 sequence discretiser: merged time grid from gradient vertices, RF sample edges and ADC times,
//      refined so that no RF-active interval exceeds dt_rf_max ("sequence-aware time
//      stepping")
//   a2 block splitter / regime classification
//   a3 k(t) table per precession block: cumulative trapezoid of G on the vertices (Eq 12-13, :173-180),
//      stored only at the points that are evaluated (ADC samples) + one end record per block
//   a4 rotation-vector table per RF step (Eq 8 with piecewise-constant B1, :146-148, :182)
#include <algorithm>
#include <cmath>
#include <cstring>
#include <atomic>
#include <limits>
#include <thread>
#include <utility>

#include "internal.h"

namespace bloch {

static thread_local std::string g_err;
void set_error(const std::string &msg) { g_err = msg; }
int fail(int code, const std::string &msg) {
    g_err = msg;
    return code;
}
const char *last_error_cstr() { return g_err.c_str(); }

namespace {

bool ascending(const double *a, int64_t n, bool strict) {
    for (int64_t i = 0; i < n; ++i) {
        if (!std::isfinite(a[i])) return false;
        if (i > 0 && (strict ? !(a[i] > a[i - 1]) : !(a[i] >= a[i - 1]))) return false;
    }
    return true;
}

// Piecewise-linear gradients of the three axes sampled on the points [n0, n1) of the (ascending) grid by a forward
// sweep: out[3 n + axis].
void sample_axes(const bloch_sequence *seq, const std::vector<double> &t, size_t n0, size_t n1, double *out) {
    for (int axis = 0; axis < 3; ++axis) {
        const double *gt = seq->g_t[axis], *gv = seq->g_v[axis];
        const int64_t gn = seq->g_n[axis];
        int64_t seg = 0;
        if (gn >= 2 && n0 < n1)  // start the sweep at the segment that holds t[n0]
            seg = std::max<int64_t>(0, std::min<int64_t>(gn - 2, (std::upper_bound(gt, gt + gn, t[n0]) - gt) - 1));
        for (size_t n = n0; n < n1; ++n) {
            double v = 0.0;
            const double tn = t[n];
            if (gn == 1) {
                v = (std::fabs(tn - gt[0]) <= kTimeTol) ? gv[0] : 0.0;
            } else if (gn >= 2 && tn >= gt[0] - kTimeTol && tn <= gt[gn - 1] + kTimeTol) {
                while (seg + 2 < gn && gt[seg + 1] <= tn) ++seg;
                const double t0 = gt[seg], t1 = gt[seg + 1];
                double w = (t1 > t0) ? (tn - t0) / (t1 - t0) : 1.0;
                w = std::min(1.0, std::max(0.0, w));
                v = gv[seg] + w * (gv[seg + 1] - gv[seg]);
            }
            out[3 * n + axis] = v;
        }
    }
}

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// fn(i) for i in [0, n) on up to `threads` host threads (items handed out in order from a shared counter).  The plan's
// blocks are independent of one another once the grid is fixed (a3, a4, table fill), and every result is written to
// the block's own slot, so the tables are the same bytes whatever the thread count.
template <class F>
void parallel_for(size_t n, unsigned threads, F fn) {
    if (threads <= 1 || n <= 1) {
        for (size_t i = 0; i < n; ++i) fn(i);
        return;
    }
    std::atomic<size_t> next{0};
    auto work = [&]() {
        for (size_t i = next.fetch_add(1); i < n; i = next.fetch_add(1)) fn(i);
    };
    std::vector<std::thread> pool;
    try {
        for (unsigned k = 1; k < threads; ++k) pool.emplace_back(work);
    } catch (...) {  // no more threads to be had: the ones that started, and this one, share the items
    }
    work();
    for (std::thread &th : pool) th.join();
}

}  // namespace

int build_plan(const bloch_scanner *scanner, const bloch_sequence *seq, const bloch_sim_params *params,
               bloch_plan *plan) {
    // ------------------------------------------------------------------ validation
    if (!seq || !params || !plan) return fail(BLOCH_EINVAL, "NULL argument");
    const double gamma = (scanner && scanner->gamma > 0.0) ? scanner->gamma : 2.0 * M_PI * 42.58e6;
    if (!std::isfinite(gamma)) return fail(BLOCH_EINVAL, "gamma not finite");
    if (!(seq->t_end > 0.0) || !std::isfinite(seq->t_end)) return fail(BLOCH_EINVAL, "t_end must be > 0");
    if (params->phase_mode < BLOCH_PHASE_AUTO || params->phase_mode > BLOCH_PHASE_FP64)
        return fail(BLOCH_EINVAL, "bad phase_mode");
    if (params->output_mode != BLOCH_OUT_SUM_ALL && params->output_mode != BLOCH_OUT_PER_SPIN &&
        params->output_mode != BLOCH_OUT_GROUPED)
        return fail(BLOCH_EINVAL, "bad output_mode");
    if (params->output_mode == BLOCH_OUT_GROUPED && params->group_size < 1)
        return fail(BLOCH_EINVAL, "group_size must be >= 1 with BLOCH_OUT_GROUPED");
    if (params->motion_mode != BLOCH_MOTION_NONE && params->motion_mode != BLOCH_MOTION_LINEAR &&
        params->motion_mode != BLOCH_MOTION_WAVEFORM)
        return fail(BLOCH_EINVAL, "bad motion_mode");
    const bool motion = params->motion_mode != BLOCH_MOTION_NONE;
    const bool waveform = params->motion_mode == BLOCH_MOTION_WAVEFORM;
    if (waveform) {
        if (params->motion_n < 1 || !params->motion_t || !params->motion_u)
            return fail(BLOCH_EINVAL, "BLOCH_MOTION_WAVEFORM needs motion_t, motion_u and motion_n >= 1");
        if (!ascending(params->motion_t, params->motion_n, true))
            return fail(BLOCH_ENONMONOTONIC, "motion waveform vertex times must be strictly ascending and finite");
        for (int64_t i = 0; i < params->motion_n; ++i)
            if (!std::isfinite(params->motion_u[i])) return fail(BLOCH_EINVAL, "motion waveform value not finite");
    }
    const double dt_mo = (motion && params->dt_max > 0.0 && std::isfinite(params->dt_max))
                             ? params->dt_max : std::numeric_limits<double>::infinity();
    for (int a = 0; a < 3; ++a) {
        if (seq->g_n[a] < 0 || (seq->g_n[a] > 0 && (!seq->g_t[a] || !seq->g_v[a])))
            return fail(BLOCH_EINVAL, "gradient arrays NULL or negative count");
        if (!ascending(seq->g_t[a], seq->g_n[a], true))
            return fail(BLOCH_ENONMONOTONIC, "gradient vertex times must be strictly ascending and finite");
        for (int64_t i = 0; i < seq->g_n[a]; ++i) {
            if (!std::isfinite(seq->g_v[a][i])) return fail(BLOCH_EINVAL, "gradient value not finite");
            if (seq->g_t[a][i] < -kTimeTol || seq->g_t[a][i] > seq->t_end + kTimeTol)
                return fail(BLOCH_EINVAL, "gradient vertex outside [0, t_end]");
        }
    }
    if (seq->rf_n < 0 || (seq->rf_n > 0 && (!seq->rf_t || !seq->rf_dt || !seq->rf_re || !seq->rf_im)))
        return fail(BLOCH_EINVAL, "RF arrays NULL or negative count");
    for (int64_t i = 0; i < seq->rf_n; ++i) {
        if (!std::isfinite(seq->rf_t[i]) || !(seq->rf_dt[i] > 0.0) || !std::isfinite(seq->rf_dt[i]) ||
            !std::isfinite(seq->rf_re[i]) || !std::isfinite(seq->rf_im[i]))
            return fail(BLOCH_EINVAL, "RF sample not finite or rf_dt <= 0");
        if (seq->rf_t[i] < -kTimeTol || seq->rf_t[i] + seq->rf_dt[i] > seq->t_end + kTimeTol)
            return fail(BLOCH_EINVAL, "RF sample outside [0, t_end]");
        if (i > 0 && seq->rf_t[i] < seq->rf_t[i - 1] + seq->rf_dt[i - 1] - kTimeTol)
            return fail(BLOCH_ENONMONOTONIC, "RF samples overlap or are not ascending");
    }
    if (seq->adc_n < 0 || (seq->adc_n > 0 && !seq->adc_t)) return fail(BLOCH_EINVAL, "ADC array NULL");
    for (int64_t i = 0; i < seq->adc_n; ++i) {
        if (!std::isfinite(seq->adc_t[i]) || seq->adc_t[i] < -kTimeTol || seq->adc_t[i] > seq->t_end + kTimeTol)
            return fail(BLOCH_EINVAL, "ADC time outside [0, t_end]");
        if (i > 0 && !(seq->adc_t[i] > seq->adc_t[i - 1] + kTimeTol))
            return fail(BLOCH_ENONMONOTONIC, "ADC times must be strictly ascending");
    }
    // hardware limits: checked when given (> 0), never part of the arithmetic.  Per axis, between
    // consecutive vertices; a waveform that starts or ends on a non-zero vertex is not charged for that edge.
    if (scanner && (scanner->G_max > 0.0 || scanner->S_max > 0.0)) {
        for (int a = 0; a < 3; ++a)
            for (int64_t i = 0; i < seq->g_n[a]; ++i) {
                if (scanner->G_max > 0.0 && std::fabs(seq->g_v[a][i]) > scanner->G_max * (1.0 + 1e-9))
                    return fail(BLOCH_EHWLIMIT, "gradient amplitude exceeds scanner G_max");
                if (scanner->S_max > 0.0 && i > 0 &&
                    std::fabs(seq->g_v[a][i] - seq->g_v[a][i - 1]) >
                        scanner->S_max * (seq->g_t[a][i] - seq->g_t[a][i - 1]) * (1.0 + 1e-9))
                    return fail(BLOCH_EHWLIMIT, "gradient slew rate exceeds scanner S_max");
            }
    }
    const double dt_rf = (params->dt_rf_max > 0.0 && std::isfinite(params->dt_rf_max))
                             ? params->dt_rf_max : std::numeric_limits<double>::infinity();
    // extents of the phantoms the plan may assume (bloch_sim_params; the plan itself never sees a spin)
    auto extent = [](double v, double dflt) { return (v > 0.0 && std::isfinite(v)) ? v : dflt; };
    if (std::isnan(params->max_extent_m) || std::isnan(params->max_offres_hz) || std::isnan(params->max_speed_mps))
        return fail(BLOCH_EINVAL, "max_extent_m / max_offres_hz / max_speed_mps is NaN");
    const double ext_m = extent(params->max_extent_m, 0.25), ext_hz = extent(params->max_offres_hz, 1000.0),
                 ext_mps = extent(params->max_speed_mps, 1.0);

    // ------------------------------------------------------------------ a1: merged grid
    // Every source is ascending on its own (validated above), so the union is a merge of sorted runs, not a sort
    // (config 5: 5.1e6 points; std::sort took half of the planning time), and the merge writes the clamped, de-duplicated
    // grid directly: small runs (end points, gradient vertices, waveform vertices) are merged into one first, then ONE
    // three-way pass over (small runs, RF sample edges, ADC times).
    std::vector<double> small_pts;
    small_pts.reserve(size_t(2 + seq->g_n[0] + seq->g_n[1] + seq->g_n[2]) + (waveform ? size_t(params->motion_n) : 0));
    small_pts.push_back(0.0);
    small_pts.push_back(seq->t_end);
    auto merge_small = [&small_pts](size_t run_first) {
        std::inplace_merge(small_pts.begin(), small_pts.begin() + (std::ptrdiff_t)run_first, small_pts.end());
    };
    for (int a = 0; a < 3; ++a) {
        const size_t first = small_pts.size();
        small_pts.insert(small_pts.end(), seq->g_t[a], seq->g_t[a] + seq->g_n[a]);
        merge_small(first);
    }
    if (waveform) {  // the vertices of the motion waveform that lie inside the sequence are points of the grid
        const size_t first = small_pts.size();
        for (int64_t i = 0; i < params->motion_n; ++i)
            if (params->motion_t[i] >= 0.0 && params->motion_t[i] <= seq->t_end) small_pts.push_back(params->motion_t[i]);
        merge_small(first);
    }
    std::vector<double> rf_pts(size_t(2 * seq->rf_n));
    for (int64_t i = 0; i < seq->rf_n; ++i) {
        rf_pts[2 * i] = seq->rf_t[i];
        rf_pts[2 * i + 1] = seq->rf_t[i] + seq->rf_dt[i];
    }
    // rf_t[i] + rf_dt[i] may exceed rf_t[i + 1] by rounding when samples abut: insertion pass over the run
    for (size_t k = 1; k < rf_pts.size(); ++k)
        for (size_t m = k; m > 0 && rf_pts[m] < rf_pts[m - 1]; --m) std::swap(rf_pts[m], rf_pts[m - 1]);
    std::vector<double> coarse;
    coarse.reserve(small_pts.size() + rf_pts.size() + size_t(seq->adc_n));
    {
        const double *pa = small_pts.data(), *ea = pa + small_pts.size();
        const double *pb = rf_pts.data(), *eb = pb + rf_pts.size();
        const double *pc = seq->adc_t, *ec = pc + seq->adc_n;
        const double inf = std::numeric_limits<double>::infinity();
        while (pa < ea || pb < eb || pc < ec) {
            const double va = pa < ea ? *pa : inf, vb = pb < eb ? *pb : inf, vc = pc < ec ? *pc : inf;
            double t;
            if (va <= vb && va <= vc) { t = va; ++pa; }
            else if (vb <= vc) { t = vb; ++pb; }
            else { t = vc; ++pc; }
            t = std::min(std::max(t, 0.0), seq->t_end);
            if (coarse.empty() || t - coarse.back() > kTimeTol) coarse.push_back(t);
        }
    }
    // RF coverage of the coarse intervals (sweep), then refinement of RF-active ones
    std::vector<double> t;          // refined points
    std::vector<int64_t> rf_of;     // per refined interval: RF sample index or -1
    t.reserve(coarse.size());
    rf_of.reserve(coarse.size());
    t.push_back(coarse[0]);
    {
        int64_t j = 0;
        for (size_t i = 0; i + 1 < coarse.size(); ++i) {
            const double a = coarse[i], b = coarse[i + 1], mid = 0.5 * (a + b);
            while (j < seq->rf_n && seq->rf_t[j] + seq->rf_dt[j] <= mid) ++j;
            const bool covered = (j < seq->rf_n && seq->rf_t[j] <= mid);
            int64_t parts = 1;
            // a piece is longer than its limit only beyond the time tolerance (readings G13 + G18); with motion
            // every interval is also limited to dt_max
            const double lim = std::min(covered ? dt_rf : std::numeric_limits<double>::infinity(), dt_mo);
            if (std::isfinite(lim)) parts = std::max<int64_t>(1, (int64_t)std::ceil(((b - a) - kTimeTol) / lim));
            for (int64_t p = 1; p <= parts; ++p) {
                t.push_back(p == parts ? b : a + (b - a) * (double(p) / double(parts)));
                rf_of.push_back(covered ? j : -1);
            }
        }
    }
    const int64_t N = (int64_t)rf_of.size();
    // motion waveform at the grid points: x(t_n) = x + a u_n; u(t) = t for constant velocities (MOTION_LINEAR), else
    // the piecewise-linear interpolant of the vertices, held at its end values outside them (forward sweep)
    std::vector<double> u(motion ? t.size() : 0);
    if (motion && !waveform) u = t;
    if (waveform) {
        const double *mt = params->motion_t, *mu = params->motion_u;
        const int64_t mn = params->motion_n;
        int64_t seg = 0;
        for (size_t n = 0; n < t.size(); ++n) {
            const double tn = t[n];
            if (tn <= mt[0]) u[n] = mu[0];
            else if (tn >= mt[mn - 1]) u[n] = mu[mn - 1];
            else {
                while (seg + 2 < mn && mt[seg + 1] <= tn) ++seg;
                u[n] = mu[seg] + (tn - mt[seg]) / (mt[seg + 1] - mt[seg]) * (mu[seg + 1] - mu[seg]);
            }
        }
    }
    // long sequences (config 5: 3.1e6 intervals, 2001 blocks) are planned on several host threads
    const unsigned n_thr = N < 200000 ? 1u : std::min(16u, std::max(1u, std::thread::hardware_concurrency()));
    std::vector<double> G(3 * t.size(), 0.0);
    {   // contiguous slices of the grid, one sweep per slice (the segment a slice starts in is found by bisection)
        const size_t n_sl = n_thr > 1 ? 4 * n_thr : 1, np = t.size();
        parallel_for(n_sl, n_thr, [&](size_t k) { sample_axes(seq, t, np * k / n_sl, np * (k + 1) / n_sl, G.data()); });
    }
    // ADC index per point (both ascending)
    std::vector<int64_t> adc_at(t.size(), -1);
    {
        size_t n = 0;
        for (int64_t i = 0; i < seq->adc_n; ++i) {
            while (n + 1 < t.size() && t[n] < seq->adc_t[i] - kTimeTol) ++n;
            if (std::fabs(t[n] - seq->adc_t[i]) > 2 * kTimeTol) return fail(BLOCH_EINVAL, "internal: ADC time not on the grid");
            if (adc_at[n] != -1) return fail(BLOCH_ENONMONOTONIC, "two ADC samples closer than 1e-12 s");
            adc_at[n] = i;
        }
    }

    // ------------------------------------------------------------------ a2: blocks
    const int64_t max_pts = params->max_block_points > 0 ? params->max_block_points : kDefaultMaxBlockPoints;
    std::vector<Block> blocks;
    {
        // An ADC sample with RF on both sides of it (strictly inside an RF run, or at t = 0 / t_end of a sequence that
        // starts / ends with RF) is served by an EMPTY precession block (no interval, tau = 0: the sample is Mxy as it
        // stands, which is what the step-by-step integrator records, reading G7) that cuts the RF run in two.
        auto empty_block = [&blocks](int64_t at) {
            Block e;
            e.type = kBlockPrecession;
            e.first = at;
            e.count = 0;
            blocks.push_back(e);
        };
        auto inside_rf = [&](int64_t n) { return n > 0 && n < N && rf_of[n - 1] >= 0 && rf_of[n] >= 0 && adc_at[n] >= 0; };
        int64_t n = 0;
        if (N > 0 && rf_of[0] >= 0 && adc_at[0] >= 0) empty_block(0);
        while (n < N) {
            Block b;
            b.type = rf_of[n] >= 0 ? kBlockRF : kBlockPrecession;
            b.first = n;
            int64_t pts_in = 0;
            while (n < N && (rf_of[n] >= 0) == (b.type == kBlockRF)) {
                if (b.type == kBlockPrecession && adc_at[n + 1] >= 0) {
                    if (pts_in + 1 > max_pts) break;
                    ++pts_in;
                }
                ++n;
                if (b.type == kBlockRF && inside_rf(n)) break;
            }
            if (n == b.first) ++n;  // max_pts == 0 guard: always advance
            b.count = n - b.first;
            blocks.push_back(b);
            if (b.type == kBlockRF && inside_rf(n)) empty_block(n);
        }
        if (N > 0 && rf_of[N - 1] >= 0 && adc_at[N] >= 0) empty_block(N);
    }
    // ADC assignment (reading G7): on an RF/precession boundary -> served by the precession block (tau = 0 or
    // tau = T); on a precession/precession cut -> the earlier; with RF on both sides -> the empty block made above.
    for (size_t bi = 0; bi < blocks.size(); ++bi) {
        Block &b = blocks[bi];
        if (b.type == kBlockRF) {
            for (int64_t n = b.first + 1; n < b.first + b.count; ++n)
                if (adc_at[n] >= 0) return fail(BLOCH_EADC_IN_RF, "internal: ADC sample left inside an RF block");
            continue;
        }
        const bool serve_start = (bi == 0) || (blocks[bi - 1].type == kBlockRF);
        const int64_t p0 = serve_start ? b.first : b.first + 1;
        b.adc_first = -1;
        b.adc_count = 0;
        for (int64_t n = p0; n <= b.first + b.count; ++n) {
            if (adc_at[n] < 0) continue;
            if (b.adc_first < 0) b.adc_first = adc_at[n];
            ++b.adc_count;
        }
        if (b.adc_first < 0) b.adc_first = 0;
    }

    // ------------------------------------------------------------------ a3 + phase-mode resolution
    const double gbar = gamma / (2.0 * M_PI);
    double worst_turns = 0.0, k_max = 0.0, tau_max = 0.0, m_max = 0.0;
    std::vector<double> krec;  // 4 doubles per evaluated point, all precession blocks in order
    std::vector<double> mrec;  // motion: (mu'x, mu'y, mu'z, 0) per evaluated point, same order
    std::vector<int64_t> krec_first(blocks.size(), 0);
    int64_t n_rf_steps = 0, n_rf_blocks = 0, n_eval = 0, max_block_adc = 0;
    {
        int64_t n_rec = 0;  // a block's records start where the blocks before it end: one per ADC sample it serves
        for (size_t bi = 0; bi < blocks.size(); ++bi) {
            const Block &b = blocks[bi];
            if (b.type == kBlockRF) {
                n_rf_steps += b.count;
                ++n_rf_blocks;
                continue;
            }
            krec_first[bi] = n_rec;
            n_rec += b.adc_count;
            n_eval += b.adc_count + 1;
            max_block_adc = std::max(max_block_adc, b.adc_count);
        }
        krec.resize(4 * (size_t)n_rec);
        if (motion) mrec.resize(4 * (size_t)n_rec);
    }
    struct A3Max { double worst = 0.0, k = 0.0, tau = 0.0, m = 0.0; };
    std::vector<A3Max> a3max(blocks.size());
    std::atomic<int> a3_bad{0};
    parallel_for(blocks.size(), n_thr, [&](size_t bi) {
        Block &b = blocks[bi];
        if (b.type == kBlockRF) return;
        A3Max &mx = a3max[bi];
        double *kr = krec.data() + 4 * krec_first[bi];
        double *mr = motion ? mrec.data() + 4 * krec_first[bi] : nullptr;
        int64_t w = 0;  // records written
        const bool serve_start = (bi == 0) || (blocks[bi - 1].type == kBlockRF);
        double K[3] = {0, 0, 0}, Mo[3] = {0, 0, 0};
        const double tb = t[b.first];
        if (serve_start && adc_at[b.first] >= 0 && w < b.adc_count) {
            for (int c = 0; c < 4; ++c) kr[c] = 0.0;
            if (motion) for (int c = 0; c < 4; ++c) mr[c] = 0.0;
            ++w;
        }
        for (int64_t n = b.first; n < b.first + b.count; ++n) {
            const double dt = t[n + 1] - t[n];
            for (int a = 0; a < 3; ++a) K[a] += 0.5 * (G[3 * n + a] + G[3 * (n + 1) + a]) * dt;  // Eq 12-13
            // motion: the same trapezoid on G(t) t, so that sum of Bz(t_n) = G_n . (x + v t_n) splits into K . x + Mo . v
            if (motion)
                for (int a = 0; a < 3; ++a) Mo[a] += 0.5 * (G[3 * n + a] * u[n] + G[3 * (n + 1) + a] * u[n + 1]) * dt;
            const double tau = t[n + 1] - tb;
            const double kn = gbar * std::sqrt(K[0] * K[0] + K[1] * K[1] + K[2] * K[2]);
            const double mn = motion ? gbar * std::sqrt(Mo[0] * Mo[0] + Mo[1] * Mo[1] + Mo[2] * Mo[2]) : 0.0;
            // |theta| <= |k'| |x| + |f| tau (+ |mu'| |v|): the bound within the declared extents, and its three
            // factors on their own for the check against the phantom a simulation is actually given (api.cu)
            mx.worst = std::max(mx.worst, kn * ext_m + ext_hz * tau + (motion ? mn * ext_mps : 0.0));
            mx.k = std::max(mx.k, kn);
            mx.tau = std::max(mx.tau, tau);
            if (motion) mx.m = std::max(mx.m, mn);
            if (adc_at[n + 1] >= 0) {
                if (w >= b.adc_count) { a3_bad.store(1); break; }
                double *q = kr + 4 * w;
                q[0] = -gbar * K[0]; q[1] = -gbar * K[1]; q[2] = -gbar * K[2]; q[3] = tau;
                if (motion) {
                    double *qm = mr + 4 * w;
                    qm[0] = -gbar * Mo[0]; qm[1] = -gbar * Mo[1]; qm[2] = -gbar * Mo[2]; qm[3] = 0.0;
                }
                ++w;
            }
        }
        for (int a = 0; a < 3; ++a) b.kend[a] = -gbar * K[a];
        for (int a = 0; a < 3; ++a) b.mend[a] = -gbar * Mo[a];
        b.tau_end = t[b.first + b.count] - tb;
        if (w != b.adc_count) a3_bad.store(1);
    });
    if (a3_bad.load()) return fail(BLOCH_EINVAL, "internal: ADC bookkeeping mismatch");
    for (const A3Max &mx : a3max) {
        worst_turns = std::max(worst_turns, mx.worst);
        k_max = std::max(k_max, mx.k);
        tau_max = std::max(tau_max, mx.tau);
        m_max = std::max(m_max, mx.m);
    }
    // AUTO: fp32 phase (in turns, block-relative) keeps ~2^-24 * turns of resolution; above 256 turns
    // (bound: |k| max_extent_m + max_offres_hz tau, + |mu'| max_speed_mps with motion) switch to fp64 phase
    // accumulation (north_star item 4).  The fp64 phase itself is a 32-bit fixed-point fraction below 2^19 turns.
    int phase = params->phase_mode;
    if (phase == BLOCH_PHASE_AUTO) phase = worst_turns > kFp32TurnLimit ? BLOCH_PHASE_FP64 : BLOCH_PHASE_FP32;
    if (phase == BLOCH_PHASE_FP64 && worst_turns >= kFp64TurnLimit)
        return fail(BLOCH_ERANGE, "a block's phase can reach 2^19 turns within the declared extents: beyond the fp64 phase path "
                                  "(shorten the blocks with max_block_points)");

    // ------------------------------------------------------------------ a4: RF tile images
    std::vector<std::vector<unsigned char>> rf_img(blocks.size());
    std::atomic<int> a4_bad{0};
    parallel_for(blocks.size(), n_thr, [&](size_t bi) {
        Block &b = blocks[bi];
        if (b.type != kBlockRF) return;
        // per step, in fp32 as the kernel sees them: rotation vector w = gamma * B * dt (Eq 8); the gradient
        // part is per metre, mean of the two vertex values (reading G5)
        struct StepF { float wx, wy, g[3], dt, h[3]; };
        std::vector<StepF> st((size_t)b.count);
        for (int64_t n = b.first; n < b.first + b.count; ++n) {
            const double dt = t[n + 1] - t[n];
            const int64_t j = rf_of[n];
            StepF &s = st[(size_t)(n - b.first)];
            s.wx = (float)(gamma * dt * seq->rf_re[j]);
            s.wy = (float)(gamma * dt * seq->rf_im[j]);
            for (int a = 0; a < 3; ++a) s.g[a] = (float)(gamma * dt * 0.5 * (G[3 * n + a] + G[3 * (n + 1) + a]));
            for (int a = 0; a < 3; ++a)
                s.h[a] = motion ? (float)(gamma * dt * 0.5 * (G[3 * n + a] * u[n] + G[3 * (n + 1) + a] * u[n + 1])) : 0.f;
            s.dt = (float)dt;
        }
        // cut into tiles: at most kRfTileSteps steps, one dt per tile
        std::vector<std::pair<size_t, size_t>> tiles;  // (first, count)
        for (size_t k = 0; k < st.size();) {
            size_t c = 1;
            while (k + c < st.size() && c < (size_t)kRfTileSteps && st[k + c].dt == st[k].dt) ++c;
            tiles.emplace_back(k, c);
            k += c;
        }
        b.n_tiles = (int64_t)tiles.size();
        const size_t dir_bytes = align_up(tiles.size() * 8, 16);
        std::vector<unsigned char> &img = rf_img[bi];
        img.assign(dir_bytes, 0);
        for (size_t ti = 0; ti < tiles.size(); ++ti) {
            const size_t k0 = tiles[ti].first, c = tiles[ti].second;
            RfTileHdr h;
            std::memset(&h, 0, sizeof(h));
            bool uniform = true;
            for (size_t k = k0; k < k0 + c; ++k) {
                const StepF &s = st[k];
                h.wxy2_max = std::max(h.wxy2_max, s.wx * s.wx + s.wy * s.wy);
                h.gx_max = std::max(h.gx_max, std::fabs(s.g[0]));
                h.gy_max = std::max(h.gy_max, std::fabs(s.g[1]));
                h.gz_max = std::max(h.gz_max, std::fabs(s.g[2]));
                uniform = uniform && s.g[0] == st[k0].g[0] && s.g[1] == st[k0].g[1] && s.g[2] == st[k0].g[2];
                if (motion) {
                    h.hx_max = std::max(h.hx_max, std::fabs(s.h[0]));
                    h.hy_max = std::max(h.hy_max, std::fabs(s.h[1]));
                    h.hz_max = std::max(h.hz_max, std::fabs(s.h[2]));
                }
            }
            if (motion) uniform = false;  // h = g t changes with every step
            h.dt = st[k0].dt;
            h.n_steps = (int32_t)c;
            h.flags = (uniform ? kRfFlagUniformG : 0) | (motion ? kRfFlagMotion : 0);
            h.gx = st[k0].g[0]; h.gy = st[k0].g[1]; h.gz = st[k0].g[2];
            const size_t rec = motion ? 48 : (uniform ? 16 : 32);
            const size_t off0 = img.size();
            img.resize(off0 + kRfHdrBytes + c * rec, 0);
            std::memcpy(img.data() + off0, &h, sizeof(h));
            float *r = reinterpret_cast<float *>(img.data() + off0 + kRfHdrBytes);
            for (size_t k = k0; k < k0 + c; ++k, r += rec / 4) {
                const StepF &s = st[k];
                r[0] = s.wx; r[1] = s.wy; r[2] = s.wx * s.wx + s.wy * s.wy; r[3] = 0.f;
                if (!uniform) { r[4] = s.g[0]; r[5] = s.g[1]; r[6] = s.g[2]; r[7] = 0.f; }
                if (motion) { r[8] = s.h[0]; r[9] = s.h[1]; r[10] = s.h[2]; r[11] = 0.f; }
            }
            int32_t *dir = reinterpret_cast<int32_t *>(img.data());
            dir[2 * ti] = (int32_t)off0;
            dir[2 * ti + 1] = (int32_t)(img.size() - off0);
        }
        if (img.size() > (size_t)INT32_MAX) a4_bad.store(1);
    });
    if (a4_bad.load()) return fail(BLOCH_EINVAL, "RF block table exceeds 2 GiB");
    // Static plans: excitation blocks whose tiles are all compact (gradient constant within the tile) and that fit ONE
    // kernel-parameter block (<= kRfConstSteps steps, <= kRfConstTiles tiles, internal.h) are packed once more for
    // rf_const_kernel.  Longer blocks keep rf_kernel: cutting them into several launches would round the hi + lo
    // state to one float at every cut, and the result would no longer be bitwise that of the other paths.
    plan->rf_const.clear();
    if (!motion) {
        for (size_t bi = 0; bi < blocks.size(); ++bi) {
            Block &b = blocks[bi];
            if (b.type != kBlockRF) continue;
            const unsigned char *tb = rf_img[bi].data();
            const int32_t *dir = reinterpret_cast<const int32_t *>(tb);
            bool compact = b.n_tiles > 0 && b.n_tiles <= kRfConstTiles && b.count <= kRfConstSteps;
            for (int64_t t = 0; t < b.n_tiles && compact; ++t) {
                RfTileHdr hd;
                std::memcpy(&hd, tb + dir[2 * t], sizeof hd);
                compact = (hd.flags & kRfFlagUniformG) && !(hd.flags & kRfFlagMotion) && hd.n_steps <= kRfConstSteps;
            }
            if (!compact) continue;
            b.rf_const_first = (int64_t)plan->rf_const.size();
            RfConstArgs cur;
            std::memset(&cur, 0, sizeof cur);
            for (int64_t t = 0; t < b.n_tiles; ++t) {
                RfTileHdr hd;
                std::memcpy(&hd, tb + dir[2 * t], sizeof hd);
                if (cur.n_tiles == kRfConstTiles || cur.n_steps + hd.n_steps > kRfConstSteps) {
                    plan->rf_const.push_back(cur);
                    std::memset(&cur, 0, sizeof cur);
                }
                RfConstTile &ct = cur.tile[cur.n_tiles++];
                ct.n_steps = hd.n_steps; ct.dt = hd.dt; ct.gx = hd.gx; ct.gy = hd.gy; ct.gz = hd.gz;
                ct.wxy2_max = hd.wxy2_max;
                std::memcpy(&cur.rec[4 * cur.n_steps], tb + dir[2 * t] + kRfHdrBytes, size_t(hd.n_steps) * 16);  // compact records
                cur.n_steps += hd.n_steps;
            }
            plan->rf_const.push_back(cur);
            b.rf_const_count = (int64_t)plan->rf_const.size() - b.rf_const_first;
        }
    }

    // ------------------------------------------------------------------ tables: layout + fill
    size_t off = 0;
    // precession records: (k', tau) per ADC sample, followed by (mu', 0) with motion
    const size_t rec_bytes = (phase == BLOCH_PHASE_FP64 ? 32 : 16) * (motion ? 2 : 1);
    parallel_for(blocks.size(), n_thr, [&](size_t bi) {
        Block &b = blocks[bi];
        // Cartesian readouts: does k' (and tau) advance by a constant step inside EVERY aligned group of 16 samples?
        // Checked on the fp64 records (turns / m): every sample within 1e-13 relative + 1e-8 turns / m (1e-13 s) of the
        // line through the group's first and last sample, the level at which the ADC times themselves are equally
        // spaced.  Such blocks go to signal_lin_kernel (signal.cuh), the n % 16 tail to signal_kernel.
        // (blocks of >= 20 groups that fill >= 60 % of the lanes of their warps: below that the per-sample kernel,
        // which gives every lane a sample, is the faster one)
        const int64_t lin_groups = b.adc_count / 16;
        if (b.type == kBlockPrecession && lin_groups >= 20 && 10 * lin_groups >= 6 * ((lin_groups + 31) / 32 * 32)) {
            const double *src = krec.data() + 4 * krec_first[bi];
            const int64_t n_g = b.adc_count / 16;
            bool ok = true;
            for (int64_t g = 0; g < n_g && ok; ++g) {
                const double *q = src + 4 * 16 * g;
                for (int c = 0; c < 4 && ok; ++c) {
                    const double a0 = q[c], a1 = q[4 * 15 + c], step = (a1 - a0) / 15.0;
                    const double tol = 1e-13 * std::max(std::fabs(a0), std::fabs(a1)) + (c == 3 ? 1e-13 : 1e-8);
                    for (int j = 1; j < 15 && ok; ++j) ok = std::fabs(q[4 * j + c] - (a0 + j * step)) <= tol;
                }
            }
            // motion: the first moment mu' must be a quadratic in the sample index (exact on a plateau): residual against
            // the parabola through samples 0, 8, 15 within 1e-13 relative + 1e-9 turns s / m
            if (motion) {
                const double *msrc = mrec.data() + 4 * krec_first[bi];
                for (int64_t g = 0; g < n_g && ok; ++g) {
                    const double *q = msrc + 4 * 16 * g;
                    for (int c = 0; c < 3 && ok; ++c) {
                        const double m0 = q[c], m8 = q[4 * 8 + c], m15 = q[4 * 15 + c];
                        const double qb = ((m15 - m0) / 15.0 - (m8 - m0) / 8.0) / 7.0, qa = (m8 - m0) / 8.0 - 8.0 * qb;
                        const double tol = 1e-13 * std::max(std::fabs(m0), std::fabs(m15)) + 1e-9;
                        for (int j = 1; j < 15 && ok; ++j) ok = std::fabs(q[4 * j + c] - (m0 + j * (qa + j * qb))) <= tol;
                    }
                }
            }
            if (ok) b.lin_pts = n_g * 16;
        }
    });
    for (size_t bi = 0; bi < blocks.size(); ++bi) {
        Block &b = blocks[bi];
        b.table_off = (int64_t)off;
        const size_t bytes = b.type == kBlockRF ? rf_img[bi].size() : size_t(b.adc_count) * rec_bytes;
        off = align_up(off + bytes, kAlign);
    }
    // whole-sequence program for the fused kernel: one SeqOp per block
    const size_t prog_off = off;
    off = align_up(off + blocks.size() * sizeof(SeqOp), kAlign);
    const size_t adcblk_off = off;
    {
        size_t n_adc_blocks = 0;
        for (const Block &b : blocks) n_adc_blocks += (b.type == kBlockPrecession && b.adc_count > 0) ? 1 : 0;
        off = align_up(off + std::max<size_t>(n_adc_blocks, 1) * sizeof(SeqAdcBlock), kAlign);
    }
    plan->tables.assign(off, 0);
    plan->prog_off = (int64_t)prog_off;
    plan->adcblk_off = (int64_t)adcblk_off;
    {
        SeqAdcBlock *ab = reinterpret_cast<SeqAdcBlock *>(plan->tables.data() + adcblk_off);
        for (const Block &b : blocks)
            if (b.type == kBlockPrecession && b.adc_count > 0) *ab++ = SeqAdcBlock{b.adc_first, (int32_t)b.adc_count, 0};
    }
    for (size_t bi = 0; bi < blocks.size(); ++bi) {
        const Block &b = blocks[bi];
        SeqOp op;
        std::memset(&op, 0, sizeof(op));
        op.type = b.type;
        op.n = (int32_t)(b.type == kBlockRF ? b.n_tiles : b.adc_count);
        op.table_off = b.table_off;
        op.adc_first = b.adc_first;
        for (int a = 0; a < 3; ++a) op.kend[a] = b.kend[a];
        op.tau_end = b.tau_end;
        std::memcpy(plan->tables.data() + prog_off + bi * sizeof(SeqOp), &op, sizeof(op));
    }
    parallel_for(blocks.size(), n_thr, [&](size_t bi) {
        const Block &b = blocks[bi];
        unsigned char *dst = plan->tables.data() + b.table_off;
        if (b.type == kBlockRF) {
            std::memcpy(dst, rf_img[bi].data(), rf_img[bi].size());
        } else {
            const double *src = krec.data() + 4 * krec_first[bi];
            const double *msrc = motion ? mrec.data() + 4 * krec_first[bi] : nullptr;
            const int stride = motion ? 8 : 4;  // scalars per point
            if (phase == BLOCH_PHASE_FP64) {
                double *r = reinterpret_cast<double *>(dst);
                for (int64_t i = 0; i < b.adc_count; ++i) {
                    for (int c = 0; c < 4; ++c) r[stride * i + c] = src[4 * i + c];
                    if (motion) for (int c = 0; c < 4; ++c) r[stride * i + 4 + c] = msrc[4 * i + c];
                }
            } else {
                // fp32 phase: k', mu' in rad (the signal kernel's phase is in radians), tau in s
                float *r = reinterpret_cast<float *>(dst);
                for (int64_t i = 0; i < b.adc_count; ++i) {
                    for (int c = 0; c < 4; ++c) r[stride * i + c] = (float)(c == 3 ? src[4 * i + c] : 2.0 * M_PI * src[4 * i + c]);
                    if (motion) for (int c = 0; c < 4; ++c) r[stride * i + 4 + c] = (float)(2.0 * M_PI * msrc[4 * i + c]);
                }
            }
        }
    });

    // ------------------------------------------------------------------ launch count (SUM_ALL, final state)
    int64_t launches = 2;  // pack + unpack
    {
        bool pending = false;
        for (const Block &b : blocks) {
            if (b.type == kBlockRF) { launches += std::max<int64_t>(1, b.rf_const_count); pending = false; continue; }
            if (pending) ++launches;
            if (b.adc_count > 0) launches += (params->output_mode == BLOCH_OUT_SUM_ALL) ? 2 : 1;
            if (params->output_mode == BLOCH_OUT_SUM_ALL && b.lin_pts > 0 && b.lin_pts < b.adc_count) ++launches;  // tail
            pending = b.count > 0;
        }
        if (pending) ++launches;
    }

    plan->gamma = gamma;
    plan->params = *params;
    plan->blocks = std::move(blocks);
    plan->n_adc_blocks = 0;
    for (const Block &b : plan->blocks) plan->n_adc_blocks += (b.type == kBlockPrecession && b.adc_count > 0) ? 1 : 0;
    plan->d_tables = nullptr;
    plan->k_max = k_max;
    plan->tau_max = tau_max;
    plan->m_max = m_max;
    plan->worst_turns = worst_turns;
    plan->ext_m = ext_m;
    plan->ext_hz = ext_hz;
    plan->ext_mps = ext_mps;
    plan->phase_requested = params->phase_mode;
    bloch_plan_info &inf = plan->info;
    inf.n_intervals = N;
    inf.n_rf_steps = n_rf_steps;
    inf.n_adc = seq->adc_n;
    inf.n_blocks = (int64_t)plan->blocks.size();
    inf.n_rf_blocks = n_rf_blocks;
    inf.n_eval_points = n_eval;
    inf.n_launches = launches;
    inf.table_bytes = (int64_t)plan->tables.size();
    inf.max_block_adc = max_block_adc;
    inf.phase_mode = phase;
    inf.output_mode = params->output_mode;
    inf.motion_mode = params->motion_mode;
    inf.group_size = params->output_mode == BLOCH_OUT_GROUPED ? params->group_size : 0;
    inf.phase_mode_requested = params->phase_mode;
    inf.path = plan->path;
    inf.max_extent_m = ext_m;
    inf.max_offres_hz = ext_hz;
    inf.max_speed_mps = ext_mps;
    inf.worst_turns = worst_turns;
    for (int k = 0; k < 16; ++k) inf.options[k] = k < BLOCH_N_OPTIONS ? plan->opt[k] : 0;
    return BLOCH_OK;
}

}  // namespace bloch

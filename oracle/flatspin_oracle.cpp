// flatspin_oracle.cpp -- TEST INFRASTRUCTURE ONLY.  Plain fp64 CPU oracle for the flatspin hot path.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may use this
// file.  It shares no code with the CUDA path (paper_2002_11401_b200/csrc) and neither includes
// the other.  It is written from /root/reference/PAPER.md (arxiv 2002.11401) and follows the
// paper's order and notation; every function cites the passage it restates.  Readings of silent /
// ambiguous passages are the ones listed in DESIGN.md ("Readings"), ids C-1..C-20, A-7.
//
//   Tier A  (orc_relax_A, orc_fields, orc_scan): the definition, step by step:
//           every iteration recomputes every h_i directly from Eq. 3 over the neighbourhood, tests
//           Eq. 5 and Eq. 6 for every spin, flips the one with the greatest left-hand side.
//   Tier B  (orc_relax_B): the same decisions with cached couplings, incrementally updated h_dip
//           (Eq. 3 is linear in s_j) and a tournament tree.  Needed where Tier A's
//           O(flips * N * K) is out of reach (configs 3-4).  Pinned by Tier A == Tier B flip logs.
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): two-dipole closed forms, lattice sums, astroid
// special cases, Philox known answers, brute-force neighbours, exhaustive <=12-spin flip orders,
// energy descent, global spin-flip symmetry, kagome 29x29 = 2638 magnets; spin-spin correlation
// and vertex populations on hand-countable states (polarised, ground state, one flipped spin); the near-tie monitor
// (note_decision / second_best / orc_monitor) against closed-form gaps of uncoupled spins, a winner placed at
// 1 +- eps, exact ties and a brute-force second maximum, in both tiers.
// Unpinned by the paper: full-config flip sequences (no published values exist); they are pinned only
// through Tier A == Tier B on small sizes plus the invariants above ("parity unpinned" for those).
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -std=c++17 -shared -fPIC flatspin_oracle.cpp -o liboracle.so
// (OpenMP only splits the per-spin loops of the two timing legs gather_cached / scan_cached over host threads.)

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

namespace {

const double NEG_INF = -std::numeric_limits<double>::infinity();

struct Params { double alpha, b, c, beta, gamma, neighbor_distance; };

// ------------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11), restated.  Reading C-11: key = (seed_lo, seed_hi),
// counter = (spin, step, stream, 0); stream 0 = thermal field.
// ------------------------------------------------------------------------------------------------
void philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
    uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
    uint32_t k0 = key_in[0], k1 = key_in[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Two independent unit normals for (seed, step, spin): Box-Muller on two 52-bit uniforms in (0,1)
// (reading C-11).  PAPER.md:67: "Two orthogonal components of the field are independently drawn from
// the Normal distribution N(0, sigma_th^2)".
void unit_normals(uint64_t seed, uint32_t step, uint32_t spin, double z[2]) {
    uint32_t ctr[4] = {spin, step, 0u, 0u};
    uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32)};
    uint32_t x[4];
    philox4x32_10(ctr, key, x);
    uint64_t a = (((uint64_t)x[0] << 32) | x[1]) >> 12;
    uint64_t b = (((uint64_t)x[2] << 32) | x[3]) >> 12;
    const double two_m52 = 1.0 / 4503599627370496.0;
    double u1 = ((double)a + 0.5) * two_m52;
    double u2 = ((double)b + 0.5) * two_m52;
    double r = std::sqrt(-2.0 * std::log(u1));
    double phi = 2.0 * M_PI * u2;
    z[0] = r * std::cos(phi);
    z[1] = r * std::sin(phi);
}

// ------------------------------------------------------------------------------------------------
// Eq. 5: left-hand side of the generalized Stoner-Wohlfarth astroid,
//   L = (|h_par| / (b h_k))^(2/gamma) + (|h_perp| / (c h_k))^(2/beta)
// Readings C-3 (absolute values), C-4 (h_k == hc[i]), C-5 (gamma on the parallel term as printed).
// ------------------------------------------------------------------------------------------------
double astroid_L(double hpar, double hperp, double hk, const Params& p) {
    double a = std::fabs(hpar) / (p.b * hk);
    double d = std::fabs(hperp) / (p.c * hk);
    return std::pow(a, 2.0 / p.gamma) + std::pow(d, 2.0 / p.beta);
}

struct Oracle {
    int64_t N = 0;
    std::vector<double> x, y, theta, ct, st, hc;
    Params p{};
    std::vector<int8_t> s;
    double sigma = 0.0; uint64_t seed = 0;
    double hx = 0.0, hy = 0.0; uint32_t step = 0;
    bool brute = false;

    // cell grid for neighbour search (host logic; pinned against brute force)
    double cell = 1.0, x0 = 0.0, y0 = 0.0; int64_t ncx = 0, ncy = 0;
    std::vector<int64_t> cell_start; std::vector<int32_t> cell_items;

    bool have_nbr = false;
    std::vector<std::vector<int32_t>> nbr;
    int64_t guard_violations = 0, coincident = 0;

    // Tier B caches
    bool have_w = false;
    std::vector<std::vector<double>> wpar, wperp;      // alpha * g_ij, field at i from nbr[i][k]
    std::vector<double> hd_par, hd_perp; bool hd_valid = false;
    std::vector<double> fx_par, fx_perp, key; std::vector<int32_t> tree; int64_t P = 1;

    // near-tie monitor
    int64_t n_events = 0; double min_gap = 1e300, min_thr = 1e300;

    // ---- neighbourhood: j != i with |r_i - r_j|^2 <= nd^2 (1 + 1e-9)  (reading A-7)
    double cut2() const { return p.neighbor_distance * p.neighbor_distance * (1.0 + 1e-9); }

    void test_pair(int64_t i, int64_t j, std::vector<int32_t>& out) {
        if (j == i) return;                                  // j != i, reading C-8
        double dx = x[i] - x[j], dy = y[i] - y[j];
        double d2 = dx * dx + dy * dy;
        double c2 = cut2();
        if (d2 == 0.0) { coincident++; return; }
        if (std::fabs(d2 / c2 - 1.0) < 1e-10) guard_violations++;
        if (d2 <= c2) out.push_back((int32_t)j);
    }

    void build_grid() {
        cell = p.neighbor_distance * (1.0 + 1e-6);
        double xmin = 1e300, ymin = 1e300, xmax = -1e300, ymax = -1e300;
        for (int64_t i = 0; i < N; ++i) {
            xmin = std::min(xmin, x[i]); xmax = std::max(xmax, x[i]);
            ymin = std::min(ymin, y[i]); ymax = std::max(ymax, y[i]);
        }
        x0 = xmin; y0 = ymin;
        ncx = (int64_t)std::floor((xmax - xmin) / cell) + 1;
        ncy = (int64_t)std::floor((ymax - ymin) / cell) + 1;
        // keep the grid small for huge cutoffs / tiny systems
        std::vector<int64_t> cnt(ncx * ncy + 1, 0);
        auto cid = [&](int64_t i) {
            int64_t cx = (int64_t)std::floor((x[i] - x0) / cell), cy = (int64_t)std::floor((y[i] - y0) / cell);
            return cy * ncx + cx;
        };
        for (int64_t i = 0; i < N; ++i) cnt[cid(i) + 1]++;
        for (size_t c = 1; c < cnt.size(); ++c) cnt[c] += cnt[c - 1];
        cell_start = cnt;
        cell_items.assign(N, 0);
        std::vector<int64_t> fill(cnt.begin(), cnt.end() - 1);
        for (int64_t i = 0; i < N; ++i) cell_items[fill[cid(i)]++] = (int32_t)i;
    }

    std::vector<int32_t> neighbors_of(int64_t i) {
        std::vector<int32_t> out;
        if (brute) {
            for (int64_t j = 0; j < N; ++j) test_pair(i, j, out);
            return out;
        }
        if (cell_start.empty()) build_grid();
        int64_t cx = (int64_t)std::floor((x[i] - x0) / cell), cy = (int64_t)std::floor((y[i] - y0) / cell);
        for (int64_t yy = std::max<int64_t>(0, cy - 1); yy <= std::min(ncy - 1, cy + 1); ++yy)
            for (int64_t xx = std::max<int64_t>(0, cx - 1); xx <= std::min(ncx - 1, cx + 1); ++xx)
                for (int64_t q = cell_start[yy * ncx + xx]; q < cell_start[yy * ncx + xx + 1]; ++q)
                    test_pair(i, cell_items[q], out);
        std::sort(out.begin(), out.end());
        return out;
    }

    int64_t build_neighbors() {
        if (!have_nbr) {
            guard_violations = 0; coincident = 0;
            nbr.resize(N);
            for (int64_t i = 0; i < N; ++i) nbr[i] = neighbors_of(i);
            have_nbr = true;
        }
        size_t K = 0;
        for (auto& r : nbr) K = std::max(K, r.size());
        return (int64_t)K;
    }

    // ---- Eq. 3: field at i from a unit moment m^_j at j, in i's fixed frame
    //      (reading C-2: parallel axis = m^_i = (cos theta_i, sin theta_i), perpendicular = (-sin, cos)).
    //      H = 3 r (m^_j . r)/|r|^5 - m^_j/|r|^3 with r = r_i - r_j.   Not yet scaled by alpha.
    void coupling(int64_t i, int64_t j, double g[2]) const {
        double dx = x[i] - x[j], dy = y[i] - y[j];
        double d2 = dx * dx + dy * dy;
        double dist = std::sqrt(d2);
        double d3 = dist * dist * dist, d5 = d3 * dist * dist;
        double dot = ct[j] * dx + st[j] * dy;
        double Hx = 3.0 * dx * dot / d5 - ct[j] / d3;
        double Hy = 3.0 * dy * dot / d5 - st[j] / d3;
        g[0] = Hx * ct[i] + Hy * st[i];
        g[1] = -Hx * st[i] + Hy * ct[i];
    }

    // h_dip,i = alpha * sum_j s_j g_ij, j ascending over the neighbourhood (Eq. 3 + PAPER.md:57)
    void hdip_direct(int64_t i, double h[2]) {
        const std::vector<int32_t>& nb = have_nbr ? nbr[i] : (tmp_nb = neighbors_of(i));
        double sp = 0.0, sq = 0.0, g[2];
        for (int32_t j : nb) { coupling(i, j, g); sp += s[j] * g[0]; sq += s[j] * g[1]; }
        h[0] = p.alpha * sp; h[1] = p.alpha * sq;
    }
    std::vector<int32_t> tmp_nb;

    // external field rotated into the local frame (Fig. 2).  PAPER.md:61: the external field
    // may be global, per-spin h_ext^(i), or a spatial vector field: here h_ext^(i) = global + local_i, summed
    // in global x,y components and then rotated (reading D-4); local_i defaults to zero.
    std::vector<double> lx, ly;
    void hext(int64_t i, double h[2]) const {
        double ex = hx, ey = hy;
        if (!lx.empty()) { ex = hx + lx[i]; ey = hy + ly[i]; }
        h[0] = ex * ct[i] + ey * st[i];
        h[1] = -ex * st[i] + ey * ct[i];
    }
    // thermal field: global x,y components sigma*(z0,z1), rotated like h_ext (C-9);
    // drawn once per (seed, step, spin) and constant during relaxation (C-10).
    void hth(int64_t i, double h[2]) const {
        if (sigma == 0.0) { h[0] = h[1] = 0.0; return; }
        double z[2]; unit_normals(seed, step, (uint32_t)i, z);
        double tx = sigma * z[0], ty = sigma * z[1];
        h[0] = tx * ct[i] + ty * st[i];
        h[1] = -tx * st[i] + ty * ct[i];
    }
    // Eq. 2: h_i = h_dip + h_ext + h_th
    void total_from_dip(int64_t i, const double d[2], double h[2]) const {
        double e[2], t[2]; hext(i, e); hth(i, t);
        h[0] = d[0] + e[0] + t[0];
        h[1] = d[1] + e[1] + t[1];
    }
    void field(int64_t i, int which, double h[2]) {
        if (which == 1) { hdip_direct(i, h); return; }
        if (which == 2) { hext(i, h); return; }
        if (which == 3) { hth(i, h); return; }
        double d[2]; hdip_direct(i, d); total_from_dip(i, d, h);
    }
    // switching key: L (Eq. 5) if Eq. 6 holds (h.m < 0  <=>  s_i h_par < 0, strict, C-6), else -inf.
    // A spin may flip iff key > 1.
    double key_of(int64_t i, const double h[2]) const {
        if (!((double)s[i] * h[0] < 0.0)) return NEG_INF;
        return astroid_L(h[0], h[1], hc[i], p);
    }

    void note_decision(double L1, double L2) {
        if (L1 > 1.0 && L2 > NEG_INF) {
            double gap = (L1 - L2) / L1;
            min_gap = std::min(min_gap, gap);
            if (gap < 1e-11) n_events++;
        }
        if (L1 > NEG_INF) {
            double thr = std::fabs(L1 - 1.0);
            min_thr = std::min(min_thr, thr);
            if (thr < 1e-11) n_events++;
        }
    }

    // ---- Tier A: one decision by the definition.  Returns flipped index or -1.
    int64_t step_A() {
        int64_t best = -1; double L1 = NEG_INF, L2 = NEG_INF;
        for (int64_t i = 0; i < N; ++i) {
            double h[2]; field(i, 0, h);
            double k = key_of(i, h);
            if (k > L1) { L2 = L1; L1 = k; best = i; }       // strict >: lowest index wins ties (C-7)
            else if (k > L2) L2 = k;
        }
        note_decision(L1, L2);
        if (!(L1 > 1.0)) return -1;                          // "greater than one", C-6
        return best;
    }
    int64_t relax_A(int64_t max_flips, int32_t* log, int64_t cap) {
        build_neighbors();
        hd_valid = false;
        int64_t n = 0;
        for (;;) {
            if (max_flips > 0 && n >= max_flips) break;
            int64_t k = step_A();
            if (k < 0) break;
            s[k] = (int8_t)-s[k];
            if (log && n < cap) log[n] = (int32_t)k;
            ++n;
        }
        return n;
    }

    // ---- Tier B
    void build_weights() {
        build_neighbors();
        if (have_w) return;
        wpar.resize(N); wperp.resize(N);
        for (int64_t i = 0; i < N; ++i) {
            wpar[i].resize(nbr[i].size()); wperp[i].resize(nbr[i].size());
            for (size_t k = 0; k < nbr[i].size(); ++k) {
                double g[2]; coupling(i, nbr[i][k], g);
                wpar[i][k] = p.alpha * g[0]; wperp[i][k] = p.alpha * g[1];
            }
        }
        have_w = true;
    }
    // (timing legs only: the loop over spins may be split over host threads; every spin's sum is unchanged)
    int nthreads = 1;
    void gather_cached() {
        build_weights();
        hd_par.assign(N, 0.0); hd_perp.assign(N, 0.0);
#pragma omp parallel for num_threads(nthreads) schedule(static)
        for (int64_t i = 0; i < N; ++i) {
            double a = 0.0, b = 0.0;
            for (size_t k = 0; k < nbr[i].size(); ++k) {
                a += s[nbr[i][k]] * wpar[i][k]; b += s[nbr[i][k]] * wperp[i][k];
            }
            hd_par[i] = a; hd_perp[i] = b;
        }
        hd_valid = true;
    }
    // Switching scan over the cached h_dip (Eq. 2 + Eqs. 5, 6 per spin): number of switchable spins and the arg-max,
    // lowest index among ties (C-7).  Same decisions as orc_scan, which recomputes Eq. 3 per pair instead.
    void scan_cached(int64_t* n_switchable, int64_t* best_index, double* best_L) {
        if (!hd_valid) gather_cached();
        const int T = nthreads > 0 ? nthreads : 1;
        std::vector<int64_t> cn(T, 0), cb(T, -1); std::vector<double> cl(T, NEG_INF);
#pragma omp parallel for num_threads(T) schedule(static, 1)
        for (int t = 0; t < T; ++t) {
            const int64_t i0 = N * t / T, i1 = N * (t + 1) / T;
            for (int64_t i = i0; i < i1; ++i) {
                double h[2]; const double d[2] = {hd_par[i], hd_perp[i]};
                total_from_dip(i, d, h);
                const double k = key_of(i, h);
                if (k > 1.0) { ++cn[t]; if (k > cl[t]) { cl[t] = k; cb[t] = i; } }
            }
        }
        int64_t n = 0, best = -1; double L1 = NEG_INF;
        for (int t = 0; t < T; ++t) { n += cn[t]; if (cl[t] > L1) { L1 = cl[t]; best = cb[t]; } }
        *n_switchable = n; *best_index = best; *best_L = best >= 0 ? L1 : NEG_INF;
    }

    bool better(int32_t a, int32_t b) const {               // key desc, index asc
        if (a < 0) return false;
        if (b < 0) return true;
        if (key[a] != key[b]) return key[a] > key[b];
        return a < b;
    }
    void recompute_key(int64_t i) {
        double h[2] = {hd_par[i] + fx_par[i], hd_perp[i] + fx_perp[i]};
        key[i] = key_of(i, h);
    }
    void tree_fix(int64_t i) {
        for (int64_t node = (P + i) >> 1; node >= 1; node >>= 1) {
            int32_t l = tree[2 * node], r = tree[2 * node + 1];
            tree[node] = better(l, r) ? l : r;
        }
    }
    double second_best(int64_t k) const {                    // best key among everything except k
        double L2 = NEG_INF;
        for (int64_t node = P + k; node > 1; node >>= 1) {
            int32_t sib = tree[node ^ 1];
            if (sib >= 0 && key[sib] > L2) L2 = key[sib];
        }
        return L2;
    }
    int64_t relax_B(int64_t max_flips, int32_t* log, int64_t cap) {
        build_weights();
        if (!hd_valid) gather_cached();
        fx_par.resize(N); fx_perp.resize(N); key.resize(N);
        P = 1; while (P < N) P <<= 1;
        tree.assign(2 * P, -1);
        for (int64_t i = 0; i < N; ++i) {
            // h_ext and h_th are constant during relaxation: cache their sum
            double e[2], t[2]; hext(i, e); hth(i, t);
            fx_par[i] = e[0] + t[0]; fx_perp[i] = e[1] + t[1];
            recompute_key(i);
            tree[P + i] = (int32_t)i;
        }
        for (int64_t node = P - 1; node >= 1; --node)
            tree[node] = better(tree[2 * node], tree[2 * node + 1]) ? tree[2 * node] : tree[2 * node + 1];
        int64_t n = 0;
        for (;;) {
            if (max_flips > 0 && n >= max_flips) break;
            int32_t k = tree[1];
            double L1 = (k >= 0) ? key[k] : NEG_INF;
            note_decision(L1, k >= 0 ? second_best(k) : NEG_INF);
            if (!(L1 > 1.0)) break;
            int8_t s_old = s[k];
            s[k] = (int8_t)-s_old;
            // linearity of Eq. 3 in s_k:  h_i -= 2 s_k,old * alpha g_ik   for every i with k in nbr(i)
            for (int32_t i : nbr[k]) {
                const std::vector<int32_t>& row = nbr[i];
                size_t pos = std::lower_bound(row.begin(), row.end(), k) - row.begin();
                hd_par[i] -= 2.0 * s_old * wpar[i][pos];
                hd_perp[i] -= 2.0 * s_old * wperp[i][pos];
                recompute_key(i); tree_fix(i);
            }
            recompute_key(k); tree_fix(k);
            if (log && n < cap) log[n] = k;
            ++n;
        }
        return n;
    }

    // ---- analysis reductions of the annealed state (section IV.B)
    // "the correlation of two spins is defined as +1 (-1) if their dipole interaction is minimized (maximized)".
    // The dipole interaction energy of the pair is E_ij = -m_i . H_ij = -s_i s_j g_par,ij (Eq. 3; the parallel
    // coupling is symmetric), so c_ij = +1 if s_i s_j g_par,ij > 0, -1 if < 0 (reading D-5).  Pairs whose
    // parallel coupling vanishes (|g_par| d^3 < 1e-9: the orientation does not change the energy) get c_ij = 0
    // and are not counted.  "as a function of their lateral separation": pairs are binned by
    // floor(|r_ij| / bin_width); every unordered pair of the neighbourhood is visited once.
    void spin_correlation(double bin_width, int64_t nbins, int64_t* sum, int64_t* count) {
        build_neighbors();
        for (int64_t b = 0; b < nbins; ++b) { sum[b] = 0; count[b] = 0; }
        for (int64_t i = 0; i < N; ++i)
            for (int32_t j : nbr[i]) {
                if (j <= i) continue;
                double dx = x[i] - x[j], dy = y[i] - y[j];
                double d = std::sqrt(dx * dx + dy * dy);
                int64_t b = (int64_t)std::floor(d / bin_width);
                if (b >= nbins) continue;
                double g[2]; coupling(i, j, g);
                if (std::fabs(g[0]) * (d * d * d) < 1e-9) continue;
                int c = ((double)s[i] * (double)s[j] * g[0] > 0.0) ? 1 : -1;
                sum[b] += c; count[b] += 1;
            }
    }

    // Vertex populations ("analysis of vertex populations"; Fig. 6: "Type I vertices"
    // have zero net magnetization, "Type II or III" a non-zero one).  A vertex is a point where four magnets meet
    // (square and pinwheel ASI); it is given by its four spin indices.  A moment points INTO the vertex if
    // m_i . (r_v - r_i) > 0, r_v = mean of the four positions.  Types by the number of moments pointing in:
    // 0 or 4 -> IV; 1 or 3 -> III; 2 -> I if the two in-pointing magnets sit on opposite sides of the vertex (the
    // net moment cancels), II if they are adjacent (net moment non-zero)  (reading D-6).
    void vertex_populations(const int32_t* vert, int64_t V, int64_t counts[4]) const {
        for (int t = 0; t < 4; ++t) counts[t] = 0;
        for (int64_t v = 0; v < V; ++v) {
            const int32_t* q = vert + 4 * v;
            double vx = 0.0, vy = 0.0;
            for (int a = 0; a < 4; ++a) { vx += x[q[a]]; vy += y[q[a]]; }
            vx *= 0.25; vy *= 0.25;
            int nin = 0; double inx = 0.0, iny = 0.0; bool first = true; bool opposite = false;
            for (int a = 0; a < 4; ++a) {
                int64_t i = q[a];
                double rx = vx - x[i], ry = vy - y[i];
                double mx = s[i] * ct[i], my = s[i] * st[i];
                if (mx * rx + my * ry > 0.0) {
                    ++nin;
                    if (first) { inx = rx; iny = ry; first = false; }
                    else opposite = (inx * rx + iny * ry) < 0.0;      // meaningful when exactly two point in
                }
            }
            int type;
            if (nin == 0 || nin == 4) type = 3;
            else if (nin == 1 || nin == 3) type = 2;
            else type = opposite ? 0 : 1;
            counts[type]++;
        }
    }

    // E = -1/2 sum_i m_i . h_dip,i - sum_i m_i . (h_ext + h_th)_i   (used by pin P-8 only; reading C-20)
    double energy() {
        double E = 0.0;
        for (int64_t i = 0; i < N; ++i) {
            double d[2], e[2], t[2]; hdip_direct(i, d); hext(i, e); hth(i, t);
            E += -0.5 * s[i] * d[0] - s[i] * (e[0] + t[0]);
        }
        return E;
    }
};

}  // namespace

extern "C" {

typedef struct { double alpha, b, c, beta, gamma, neighbor_distance; } orc_params;

void* orc_create(int64_t N, const double* pos, const double* angle, const double* hc,
                 const orc_params* p, int brute_force_neighbors) {
    Oracle* o = new Oracle();
    o->N = N;
    o->x.resize(N); o->y.resize(N); o->theta.assign(angle, angle + N); o->hc.assign(hc, hc + N);
    o->ct.resize(N); o->st.resize(N);
    for (int64_t i = 0; i < N; ++i) {
        o->x[i] = pos[2 * i]; o->y[i] = pos[2 * i + 1];
        o->ct[i] = std::cos(angle[i]); o->st[i] = std::sin(angle[i]);
    }
    o->p = Params{p->alpha, p->b, p->c, p->beta, p->gamma, p->neighbor_distance};
    o->s.assign(N, 1);
    o->brute = brute_force_neighbors != 0;
    return o;
}
void orc_destroy(void* h) { delete (Oracle*)h; }
int64_t orc_build_neighbors(void* h) { return ((Oracle*)h)->build_neighbors(); }
int64_t orc_guard_violations(void* h) { return ((Oracle*)h)->guard_violations; }
int64_t orc_coincident(void* h) { return ((Oracle*)h)->coincident; }
int64_t orc_num_interactions(void* h) {
    Oracle* o = (Oracle*)h; o->build_neighbors();
    int64_t I = 0; for (auto& r : o->nbr) I += (int64_t)r.size(); return I;
}
void orc_get_neighbors(void* h, int32_t* out, int64_t K) {
    Oracle* o = (Oracle*)h; o->build_neighbors();
    for (int64_t i = 0; i < o->N; ++i)
        for (int64_t k = 0; k < K; ++k) out[i * K + k] = k < (int64_t)o->nbr[i].size() ? o->nbr[i][k] : -1;
}
int64_t orc_neighbors_of(void* h, int64_t i, int32_t* out, int64_t cap) {
    Oracle* o = (Oracle*)h;
    std::vector<int32_t> nb = o->have_nbr ? o->nbr[i] : o->neighbors_of(i);
    for (int64_t k = 0; k < (int64_t)nb.size() && k < cap; ++k) out[k] = nb[k];
    return (int64_t)nb.size();
}
void orc_set_spins(void* h, const int8_t* s) { Oracle* o = (Oracle*)h; o->s.assign(s, s + o->N); o->hd_valid = false; }
void orc_get_spins(void* h, int8_t* s) { Oracle* o = (Oracle*)h; std::memcpy(s, o->s.data(), o->N); }
void orc_set_thermal(void* h, double sigma, uint64_t seed) { Oracle* o = (Oracle*)h; o->sigma = sigma; o->seed = seed; }
void orc_set_local_field(void* h, const double* hl /*[N,2] or NULL*/) {
    Oracle* o = (Oracle*)h;
    o->lx.clear(); o->ly.clear();
    if (hl) { o->lx.resize(o->N); o->ly.resize(o->N); for (int64_t i = 0; i < o->N; ++i) { o->lx[i] = hl[2 * i]; o->ly[i] = hl[2 * i + 1]; } }
}
void orc_set_field(void* h, double hx, double hy, uint32_t step) { Oracle* o = (Oracle*)h; o->hx = hx; o->hy = hy; o->step = step; }
void orc_coupling(void* h, int64_t i, int64_t j, double* g) { ((Oracle*)h)->coupling(i, j, g); }
void orc_field_one(void* h, int64_t i, int which, double* out) { ((Oracle*)h)->field(i, which, out); }
void orc_fields(void* h, int which, double* out) {
    Oracle* o = (Oracle*)h; if (which <= 1) o->build_neighbors();
    for (int64_t i = 0; i < o->N; ++i) o->field(i, which, out + 2 * i);
}
double orc_key_one(void* h, int64_t i) { Oracle* o = (Oracle*)h; double f[2]; o->field(i, 0, f); return o->key_of(i, f); }
void orc_scan(void* h, int64_t* n_switchable, int64_t* best_index, double* best_L) {
    Oracle* o = (Oracle*)h; o->build_neighbors();
    int64_t n = 0, best = -1; double L1 = NEG_INF;
    for (int64_t i = 0; i < o->N; ++i) {
        double f[2]; o->field(i, 0, f);
        double k = o->key_of(i, f);
        if (k > 1.0) { ++n; if (k > L1) { L1 = k; best = i; } }
    }
    *n_switchable = n; *best_index = best; *best_L = (best >= 0) ? L1 : NEG_INF;
}
int64_t orc_relax_A(void* h, int64_t max_flips, int32_t* log, int64_t cap) { return ((Oracle*)h)->relax_A(max_flips, log, cap); }
int64_t orc_relax_B(void* h, int64_t max_flips, int32_t* log, int64_t cap) { return ((Oracle*)h)->relax_B(max_flips, log, cap); }
void orc_cached_hdip(void* h, double* out) {
    Oracle* o = (Oracle*)h; if (!o->hd_valid) o->gather_cached();
    for (int64_t i = 0; i < o->N; ++i) { out[2 * i] = o->hd_par[i]; out[2 * i + 1] = o->hd_perp[i]; }
}
void orc_gather_cached(void* h) { ((Oracle*)h)->gather_cached(); }
void orc_set_threads(void* h, int n) { ((Oracle*)h)->nthreads = n > 0 ? n : 1; }
void orc_build_weights(void* h) { ((Oracle*)h)->build_weights(); }
void orc_scan_cached(void* h, int64_t* n_switchable, int64_t* best_index, double* best_L) {
    ((Oracle*)h)->scan_cached(n_switchable, best_index, best_L);
}
void orc_monitor(void* h, int64_t* n_events, double* min_gap, double* min_thr, int reset) {
    Oracle* o = (Oracle*)h; *n_events = o->n_events; *min_gap = o->min_gap; *min_thr = o->min_thr;
    if (reset) { o->n_events = 0; o->min_gap = 1e300; o->min_thr = 1e300; }
}
void orc_spin_correlation(void* h, double bin_width, int64_t nbins, int64_t* sum, int64_t* count) {
    ((Oracle*)h)->spin_correlation(bin_width, nbins, sum, count);
}
void orc_vertex_populations(void* h, const int32_t* vert, int64_t V, int64_t* counts4) {
    ((Oracle*)h)->vertex_populations(vert, V, counts4);
}
double orc_energy(void* h) { Oracle* o = (Oracle*)h; o->build_neighbors(); return o->energy(); }
double orc_astroid_L(double hpar, double hperp, double hk, const orc_params* p) {
    Params q{p->alpha, p->b, p->c, p->beta, p->gamma, p->neighbor_distance};
    return astroid_L(hpar, hperp, hk, q);
}
void orc_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }
void orc_unit_normals(uint64_t seed, uint32_t step, uint32_t spin, double* z) { unit_normals(seed, step, spin, z); }

}  // extern "C"

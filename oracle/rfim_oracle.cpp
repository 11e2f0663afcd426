// rfim_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded (optionally replica-parallel, bit-identical) CPU
// oracle for the hot path of Exchange Monte Carlo (parallel tempering) on the 3D
// Random Field Ising Model, written from the paper (arxiv 1508.06268, PAPER.md)
// and from the readings listed in DESIGN.md section 3 ("Readings").  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// build, link or call this file.  It shares no code with the CUDA path under
// paper_1508_06268_b200/csrc/.
//
// What follows the paper, passage by passage:
//   Hamiltonian           H = -J sum_<ij> s_i s_j - h sum_i h_i s_i      PAPER.md:25  (Eq. 1)
//   PT main loop          steps 1-4 of section 3.1
//   exchange acceptance   W = min(1, e^Delta),
//                         Delta = (beta_{i+1}-beta_i)(H(X_{i+1})-H(X_i))  PAPER.md:72-75 (Eq. 2; reading G1)
//   odd xor even pairs    j-th exchange odd/even                          PAPER.md:70,75 (reading G3)
//   checkerboard colour   A = (x+y+z) mod 2                               PAPER.md:101 (Eq. 3)
//   temperature swap      two index arrays replica<->temperature          PAPER.md:131-137 (reading G2)
//   adaptation            lowest-rate intervals get a midpoint T          PAPER.md:147-153 (readings G5,G6,G10)
//   magnetisation         |1/V sum s_i|                                    PAPER.md:251 (Eq. 11)
//   specific heat, Binder C = L^3/T^2 (<e^2>-<e>^2), g = (3 - [<M^4>]/[<M^2>]^2)/2  PAPER.md:253-260 (Eq. 12-13)
// What the paper is silent on and north_star (BASELINE.json) fixes: Philox4x32-10
// random numbers keyed on (seed, replica, sweep, site), and the acceptance
// thresholds floor(min(1, exp(-dE/T)) * 2^32) compared against one 32-bit word.
//
// Parity pins: see tests/test_oracle_*.py.  "parity unpinned" (fixed only by
// DESIGN.md, enforced only as oracle == CUDA): the prune half of the fixed-R
// adaptation rule, the spins given to an inserted replica, the Philox counter
// layout, and which colour is swept first.
//
// Build: g++ -O3 -std=c++17 -ffp-contract=off -fPIC -shared [-fopenmp] (see oracle/build.py)

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>
#include <algorithm>

namespace {

// ---------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  One call maps a 128-bit
// counter and a 64-bit key to four 32-bit words.  Ten rounds; the key is bumped
// by the Weyl constants between rounds.
// ---------------------------------------------------------------------------
void philox4x32_10(const uint32_t key_in[2], const uint32_t ctr_in[4], uint32_t out[4]) {
    const uint32_t MUL0 = 0xD2511F53u, MUL1 = 0xCD9E8D57u;
    const uint32_t WEYL0 = 0x9E3779B9u, WEYL1 = 0xBB67AE85u;
    uint32_t k0 = key_in[0], k1 = key_in[1];
    uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += WEYL0; k1 += WEYL1; }
        const uint64_t p0 = (uint64_t)MUL0 * (uint64_t)c0;
        const uint64_t p1 = (uint64_t)MUL1 * (uint64_t)c2;
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n1 = lo1;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        const uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Counter domains (reading S2): word 3 of the counter.
enum : uint32_t { DOM_COLOUR0 = 0, DOM_COLOUR1 = 1, DOM_EXCHANGE = 2, DOM_INIT_SPINS = 3, DOM_FIELD = 4 };

const double TWO32 = 4294967296.0;
const double FIELD_SCALE = 1048576.0;        // 2^20: Gaussian field is g_i * 2^-20
const int32_t FIELD_CLAMP = 8 * 1048576;     // |g_i| <= 8 * 2^20

// north_star: threshold = floor(min(1, exp(-x)) * 2^32) with x = dE * beta.  Kept as a
// 33-bit integer in [0, 2^32]; a 32-bit word u is accepted iff u < threshold.
uint64_t threshold_from_x(double x) {
    const double p = std::exp(-x);
    if (p >= 1.0) return (uint64_t)1 << 32;
    return (uint64_t)std::floor(p * TWO32);
}

struct Measurement { int64_t Eb, Ef, Msum; };

// The planning step of the adaptation (PAPER.md:147-153 + DESIGN.md reading S8), as a pure function of the ladder and
// the trial's exchange rates: which intervals get their midpoint temperature (split[t], t = 0..n-2) and, in the fixed-count
// mode (n == R), which ranks are given up (removed[u]).  Oracle::adapt applies it; the tests call it directly with
// hand-built rate vectors.
static void plan_ladder(const std::vector<double>& T, const std::vector<double>& rate, int n, int R, int insertions,
                        std::vector<char>& split, std::vector<char>& removed) {
    (void)T;
    split.assign(n > 1 ? n - 1 : 0, 0);
    removed.assign(n, 0);
    // the a lowest-rate intervals, ties broken by lower t (the paper's min-heap pops)
    std::vector<int> order(n - 1);
    for (int t = 0; t < n - 1; ++t) order[t] = t;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return rate[a] < rate[b]; });
    if (n < R) {
        // paper rule: insert midpoints, replica count grows
        const int a = std::min(std::min(insertions, R - n), n - 1);
        for (int q = 0; q < a; ++q) split[order[q]] = 1;
        return;
    }
    // fixed-R rule (reading G10): insert-and-prune, rank preserving
    const int a = std::min(insertions, n - 1);
    if (a < 1) return;
    std::vector<char> inS(n - 1, 0);
    std::vector<int> S;
    for (int q = 0; q < a; ++q) { inS[order[q]] = 1; S.push_back(order[q]); }
    // rho = the largest rate among the intervals to be split.  Removing rank u merges intervals
    // u-1 and u; its rate is predicted (conservatively) as r1*r2*min(r1,r2); u is eligible only
    // if that prediction stays above rho, so a move never creates an interval worse than those it fixes.
    const double rho = rate[S.back()];
    auto score = [&](int u) {
        const double r1 = rate[u - 1], r2 = rate[u];
        return (r1 * r2) * std::min(r1, r2);
    };
    std::vector<int> cand;
    for (int u = 1; u <= n - 2; ++u)
        if (!inS[u - 1] && !inS[u] && score(u) > rho) cand.push_back(u);
    // highest score first, ties broken by larger u
    std::stable_sort(cand.begin(), cand.end(), [&](int p, int q) {
        if (score(p) != score(q)) return score(p) > score(q);
        return p > q;
    });
    int n_removed = 0;
    for (int u : cand) {
        if (n_removed == a) break;
        if (removed[u - 1] || removed[u + 1]) continue;   // never two adjacent
        removed[u] = 1;
        n_removed += 1;
    }
    for (int q = 0; q < n_removed; ++q) split[S[q]] = 1;  // shrink the insertions if candidates ran out
}

struct Oracle {
    int L = 0, R = 0, n = 0, kind = 0;       // R = capacity (slots), n = active temperatures
    int64_t N = 0;
    double J = 0, h = 0;
    uint32_t key[2] = {0, 0};
    std::vector<std::vector<int8_t>> spins;  // [slot][i], +-1, i = x + L*(y + L*z)
    std::vector<int8_t> hb;                  // bimodal field +-1
    std::vector<int32_t> g;                  // Gaussian field, fixed point 2^-20
    std::vector<double> T, beta;             // by temperature rank
    std::vector<int32_t> t2r, r2t;           // rank -> slot, slot -> rank (-1 if inactive)
    std::vector<uint64_t> thr_bimodal;       // [rank][k][b], k = (s*n+6)/2, b = (s*h_i+1)/2
    uint64_t sweep_g = 0, xstep = 0;         // global sweep index, global exchange-step index
    std::vector<uint64_t> att, acc;          // per adjacent pair (lower rank)
    std::vector<Measurement> series;         // [step][rank]
    int64_t series_steps = 0;
    int last_exchange_every = 10;            // PAPER.md:224 "10 Metropolis sweeps"
    int insertions = 4;                      // PAPER.md:151 Fig. 6 "lowest four"
    int threads = 1;
    bool have_T = false;
    std::string err;

    inline int64_t idx(int x, int y, int z) const { return x + (int64_t)L * (y + (int64_t)L * z); }
    inline int wrap(int a) const { return a < 0 ? a + L : (a >= L ? a - L : a); }

    int neighbour_sum(const std::vector<int8_t>& s, int x, int y, int z) const {
        // six periodic neighbours; for L = 2 the +1 and -1 neighbour coincide and both count
        return s[idx(wrap(x + 1), y, z)] + s[idx(wrap(x - 1), y, z)]
             + s[idx(x, wrap(y + 1), z)] + s[idx(x, wrap(y - 1), z)]
             + s[idx(x, y, wrap(z + 1))] + s[idx(x, y, wrap(z - 1))];
    }

    // energy change of flipping site i with spin s, neighbour sum nsum: dE = 2 s (J n + h h_i)
    double delta_e(int s, int nsum, int64_t i) const {
        if (kind == 0) {
            return 2.0 * (double)s * (J * (double)nsum + h * (double)hb[i]);
        } else {
            const double hq = h / FIELD_SCALE;                 // exact: power-of-two scaling
            return 2.0 * (double)s * (J * (double)nsum + hq * (double)g[i]);
        }
    }

    uint64_t site_threshold(int slot, int x, int y, int z) const {
        const std::vector<int8_t>& s = spins[slot];
        const int64_t i = idx(x, y, z);
        const int rank = r2t[slot];
        const int nsum = neighbour_sum(s, x, y, z);
        if (kind == 0) {
            const int k = (s[i] * nsum + 6) / 2;
            const int b = (s[i] * hb[i] + 1) / 2;
            return thr_bimodal[(size_t)rank * 14 + k * 2 + b];
        }
        const double dE = delta_e(s[i], nsum, i);
        return threshold_from_x(dE * beta[rank]);
    }

    // one checkerboard half-sweep of one replica slot (Eq. 3: A = (x+y+z) mod 2)
    void half_sweep(int slot, int colour, uint64_t sweep_index) {
        std::vector<int8_t>& s = spins[slot];
        const int Lh = L / 2;
        uint32_t words[4] = {0, 0, 0, 0};
        uint64_t words_call = ~(uint64_t)0;      // which Philox call `words` holds (4 consecutive j share one)
        for (int z = 0; z < L; ++z)
            for (int y = 0; y < L; ++y)
                for (int xh = 0; xh < Lh; ++xh) {
                    const int x = 2 * xh + ((y + z + colour) & 1);
                    // j = index of this site among the sites of its colour
                    const uint64_t j = (uint64_t)xh + (uint64_t)Lh * ((uint64_t)y + (uint64_t)L * z);
                    if ((j >> 2) != words_call) {
                        const uint32_t ctr[4] = {(uint32_t)(j >> 2), (uint32_t)sweep_index, (uint32_t)slot,
                                                 colour == 0 ? DOM_COLOUR0 : DOM_COLOUR1};
                        philox4x32_10(key, ctr, words);
                        words_call = j >> 2;
                    }
                    const uint32_t u = words[j & 3];
                    const uint64_t thr = site_threshold(slot, x, y, z);
                    if ((uint64_t)u < thr) s[idx(x, y, z)] = (int8_t)(-s[idx(x, y, z)]);
                }
    }

    void sweep_slot(int slot, uint64_t sweep_index) {
        half_sweep(slot, 0, sweep_index);    // reading G4: colour A = 0 first
        half_sweep(slot, 1, sweep_index);
    }

    // Eb = sum over the 3N bonds (i,i+x),(i,i+y),(i,i+z) of s_i s_j ; Ef = sum h_i s_i (or g_i s_i) ; Msum = sum s_i
    Measurement measure_slot(int slot) const {
        const std::vector<int8_t>& s = spins[slot];
        Measurement m{0, 0, 0};
        for (int z = 0; z < L; ++z)
            for (int y = 0; y < L; ++y)
                for (int x = 0; x < L; ++x) {
                    const int64_t i = idx(x, y, z);
                    const int si = s[i];
                    m.Eb += si * (s[idx(wrap(x + 1), y, z)] + s[idx(x, wrap(y + 1), z)] + s[idx(x, y, wrap(z + 1))]);
                    m.Ef += (kind == 0) ? (int64_t)si * hb[i] : (int64_t)si * g[i];
                    m.Msum += si;
                }
        return m;
    }

    // E = -J*Eb - hs*Ef  (Eq. 1), evaluated as (-J*Eb) - (hs*Ef) in binary64
    double energy_of(const Measurement& m) const {
        const double hs = (kind == 0) ? h : h / FIELD_SCALE;
        const double t1 = -J * (double)m.Eb;
        const double t2 = hs * (double)m.Ef;
        return t1 - t2;
    }

    void rebuild_tables() {
        beta.resize(n);
        for (int t = 0; t < n; ++t) beta[t] = 1.0 / T[t];
        if (kind == 0) {
            thr_bimodal.assign((size_t)n * 14, 0);
            for (int t = 0; t < n; ++t)
                for (int k = 0; k <= 6; ++k)
                    for (int b = 0; b <= 1; ++b) {
                        const double dE = 2.0 * (J * (double)(2 * k - 6) + h * (double)(2 * b - 1));
                        thr_bimodal[(size_t)t * 14 + k * 2 + b] = threshold_from_x(dE * beta[t]);
                    }
        }
    }

    void reset_statistics() {
        att.assign(R > 1 ? R - 1 : 0, 0);
        acc.assign(R > 1 ? R - 1 : 0, 0);
        series.clear();
        series_steps = 0;
    }

    // one exchange step: measure, then odd xor even adjacent pairs
    void exchange_step() {
        std::vector<Measurement> m(n);
        std::vector<double> E(n);
        for (int t = 0; t < n; ++t) {
            m[t] = measure_slot(t2r[t]);
            E[t] = energy_of(m[t]);
            series.push_back(m[t]);
        }
        series_steps += 1;
        for (int t = (int)(xstep & 1); t + 1 <= n - 1; t += 2) {
            const double delta = (beta[t + 1] - beta[t]) * (E[t + 1] - E[t]);
            att[t] += 1;
            bool accept;
            if (delta >= 0.0) {
                accept = true;
            } else {
                const uint32_t ctr[4] = {(uint32_t)t, (uint32_t)xstep, 0u, DOM_EXCHANGE};
                uint32_t w[4];
                philox4x32_10(key, ctr, w);
                const uint64_t thr = (uint64_t)std::floor(std::exp(delta) * TWO32);
                accept = (uint64_t)w[0] < thr;
            }
            if (accept) {
                const int a = t2r[t], b = t2r[t + 1];
                t2r[t] = b; t2r[t + 1] = a;
                r2t[b] = t; r2t[a] = t + 1;
                acc[t] += 1;
            }
        }
        xstep += 1;
    }

    int do_sweeps(int64_t n_sweeps, int exchange_every) {
        if (!have_T) { err = "temperatures not set"; return -2; }
        if (n_sweeps < 0 || exchange_every < 0) { err = "bad argument"; return -1; }
        if (exchange_every > 0) last_exchange_every = exchange_every;
        for (int64_t it = 0; it < n_sweeps; ++it) {
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads)
#endif
            for (int t = 0; t < n; ++t) sweep_slot(t2r[t], sweep_g);
            sweep_g += 1;
            if (exchange_every > 0 && (sweep_g % (uint64_t)exchange_every) == 0) exchange_step();
        }
        return 0;
    }

    // Adaptation (PAPER.md:147-153 + DESIGN.md reading S8).  One trial run, then one update.
    int adapt(int64_t trial_sweeps) {
        if (!have_T) { err = "temperatures not set"; return -2; }
        reset_statistics();
        int rc = do_sweeps(trial_sweeps, last_exchange_every);
        if (rc) return rc;
        std::vector<double> rate(n - 1);
        for (int t = 0; t < n - 1; ++t) {
            if (att[t] == 0) { err = "no exchange attempts in trial"; return -2; }
            rate[t] = (double)acc[t] / (double)att[t];
        }
        std::vector<char> split, removed;
        plan_ladder(T, rate, n, R, insertions, split, removed);
        std::vector<double> newT;
        std::vector<int32_t> new_t2r;
        if (n < R) {
            // paper rule: insert midpoints, replica count grows
            int next_slot = n;                               // slots n..R-1 are the pre-allocated pool
            for (int t = 0; t < n; ++t) {
                newT.push_back(T[t]);
                new_t2r.push_back(t2r[t]);
                if (t < n - 1 && split[t]) {
                    newT.push_back((T[t] + T[t + 1]) / 2.0);     // reading G5: midpoint in T
                    spins[next_slot] = spins[t2r[t]];         // reading G6: copy the colder neighbour
                    new_t2r.push_back(next_slot);
                    next_slot += 1;
                }
            }
        } else {
            // fixed-R rule (reading G10): insert-and-prune, rank preserving
            for (int t = 0; t < n; ++t) {
                if (!removed[t]) newT.push_back(T[t]);
                if (t < n - 1 && split[t]) newT.push_back((T[t] + T[t + 1]) / 2.0);
            }
            new_t2r = t2r;                                    // slot at rank j keeps rank j: no lattice moves
            new_t2r.resize(n);
        }
        n = (int)newT.size();
        T = newT;
        t2r.assign(R, -1);
        r2t.assign(R, -1);
        for (int t = 0; t < n; ++t) { t2r[t] = new_t2r[t]; r2t[new_t2r[t]] = t; }
        rebuild_tables();
        reset_statistics();
        return 0;
    }
};

void generate_field(Oracle& o) {
    const int64_t N = o.N;
    if (o.kind == 0) o.hb.assign(N, 0); else o.g.assign(N, 0);
    for (int64_t i = 0; i < N; ++i) {
        const uint32_t ctr[4] = {(uint32_t)i, 0u, 0u, DOM_FIELD};
        uint32_t w[4];
        philox4x32_10(o.key, ctr, w);
        if (o.kind == 0) {
            o.hb[i] = (w[0] >> 31) ? (int8_t)1 : (int8_t)-1;        // h_i = rand(+-1)
        } else {
            // Box-Muller in binary64 (BASELINE.json configs 2,4,5; not in the paper)
            const double u1 = ((double)w[0] + 1.0) / TWO32;
            const double u2 = (double)w[1] / TWO32;
            const double zz = std::sqrt(-2.0 * std::log(u1)) * std::cos(6.283185307179586476925286766559 * u2);
            long long q = std::llrint(zz * FIELD_SCALE);
            if (q > FIELD_CLAMP) q = FIELD_CLAMP;
            if (q < -FIELD_CLAMP) q = -FIELD_CLAMP;
            o.g[i] = (int32_t)q;
        }
    }
}

void generate_spins(Oracle& o) {
    for (int r = 0; r < o.R; ++r) {
        o.spins[r].assign(o.N, 0);
        for (int64_t i = 0; i < o.N; ++i) {
            const uint32_t ctr[4] = {(uint32_t)(i >> 2), 0u, (uint32_t)r, DOM_INIT_SPINS};
            uint32_t w[4];
            philox4x32_10(o.key, ctr, w);
            o.spins[r][i] = (w[i & 3] >> 31) ? (int8_t)1 : (int8_t)-1;
        }
    }
}

}  // namespace

extern "C" {

void oracle_philox4x32_10(uint32_t k0, uint32_t k1, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t* out4) {
    const uint32_t key[2] = {k0, k1};
    const uint32_t ctr[4] = {c0, c1, c2, c3};
    philox4x32_10(key, ctr, out4);
}

uint64_t oracle_threshold_from_x(double x) { return threshold_from_x(x); }

int oracle_create(void** out, int L, int R, double J, double h, int field_kind, uint64_t seed) {
    if (!out || L < 2 || (L & 1) || R < 1 || (field_kind != 0 && field_kind != 1)) return -1;
    Oracle* o = new Oracle();
    o->L = L; o->R = R; o->J = J; o->h = h; o->kind = field_kind;
    o->N = (int64_t)L * L * L;
    o->key[0] = (uint32_t)(seed & 0xFFFFFFFFull);
    o->key[1] = (uint32_t)(seed >> 32);
    o->spins.resize(R);
    generate_field(*o);
    generate_spins(*o);
    o->t2r.assign(R, -1);
    o->r2t.assign(R, -1);
    o->reset_statistics();
    *out = o;
    return 0;
}

int oracle_destroy(void* p) { delete (Oracle*)p; return 0; }

int oracle_set_threads(void* p, int threads) { ((Oracle*)p)->threads = threads < 1 ? 1 : threads; return 0; }

int oracle_set_temperatures(void* p, const double* T, int n) {
    Oracle* o = (Oracle*)p;
    if (!T || n < 1 || n > o->R) return -1;
    for (int t = 0; t < n; ++t) {
        if (!(T[t] > 0.0)) return -1;
        if (t > 0 && !(T[t] > T[t - 1])) return -1;
    }
    o->n = n;
    o->T.assign(T, T + n);
    o->t2r.assign(o->R, -1);
    o->r2t.assign(o->R, -1);
    for (int t = 0; t < n; ++t) { o->t2r[t] = t; o->r2t[t] = t; }   // step 3: X_i <- beta_i
    o->rebuild_tables();
    o->reset_statistics();
    o->have_T = true;
    return 0;
}

int oracle_sweep(void* p, int64_t n_sweeps, int exchange_every) { return ((Oracle*)p)->do_sweeps(n_sweeps, exchange_every); }

int oracle_adapt_temperatures(void* p, int64_t trial_sweeps) { return ((Oracle*)p)->adapt(trial_sweeps); }

// The planning step alone (no state): new ladder for ladder T[n] with interval rates rate[n-1], capacity R, a insertions.
// out_T has room for R values; returns the new count in *out_n.  Inserted temperatures are midpoints (reading G5).
int oracle_plan_adaptation(const double* T, const double* rate, int n, int R, int a, double* out_T, int* out_n) {
    if (!T || !rate || !out_T || !out_n || n < 2 || n > R) return -1;
    std::vector<double> Tv(T, T + n), rv(rate, rate + n - 1);
    std::vector<char> split, removed;
    plan_ladder(Tv, rv, n, R, a, split, removed);
    int m = 0;
    for (int t = 0; t < n; ++t) {
        if (!removed[t]) out_T[m++] = Tv[t];
        if (t < n - 1 && split[t]) out_T[m++] = (Tv[t] + Tv[t + 1]) / 2.0;
    }
    *out_n = m;
    return 0;
}

int oracle_set_adapt_params(void* p, int exchange_every, int insertions) {
    Oracle* o = (Oracle*)p;
    if (exchange_every < 1 || insertions < 1) return -1;
    o->last_exchange_every = exchange_every;
    o->insertions = insertions;
    return 0;
}

// E[t] = H of the replica now at rank t; M[t] = (1/N) sum s_i; rate[t] = acc/att of pair (t,t+1), -1 if att = 0
int oracle_observables(void* p, double* E, double* M, double* rate) {
    Oracle* o = (Oracle*)p;
    if (!o->have_T) return -2;
    for (int t = 0; t < o->n; ++t) {
        const Measurement m = o->measure_slot(o->t2r[t]);
        if (E) E[t] = o->energy_of(m);
        if (M) M[t] = (double)m.Msum / (double)o->N;
    }
    if (rate)
        for (int t = 0; t < o->n - 1; ++t)
            rate[t] = o->att[t] ? (double)o->acc[t] / (double)o->att[t] : -1.0;
    return 0;
}

int oracle_get_spins(void* p, int temp_rank, int8_t* out) {
    Oracle* o = (Oracle*)p;
    if (!o->have_T || temp_rank < 0 || temp_rank >= o->n) return -1;
    std::memcpy(out, o->spins[o->t2r[temp_rank]].data(), (size_t)o->N);
    return 0;
}

// ---- test-only accessors -------------------------------------------------
int oracle_get_spins_slot(void* p, int slot, int8_t* out) {
    Oracle* o = (Oracle*)p;
    if (slot < 0 || slot >= o->R) return -1;
    std::memcpy(out, o->spins[slot].data(), (size_t)o->N);
    return 0;
}
int oracle_set_spins_slot(void* p, int slot, const int8_t* in) {
    Oracle* o = (Oracle*)p;
    if (slot < 0 || slot >= o->R) return -1;
    for (int64_t i = 0; i < o->N; ++i) if (in[i] != 1 && in[i] != -1) return -1;
    o->spins[slot].assign(in, in + o->N);
    return 0;
}
// field as int32: bimodal +-1, Gaussian g_i (units of 2^-20)
int oracle_get_field(void* p, int32_t* out) {
    Oracle* o = (Oracle*)p;
    for (int64_t i = 0; i < o->N; ++i) out[i] = o->kind == 0 ? (int32_t)o->hb[i] : o->g[i];
    return 0;
}
int oracle_set_field(void* p, const int32_t* in) {
    Oracle* o = (Oracle*)p;
    for (int64_t i = 0; i < o->N; ++i) {
        if (o->kind == 0) { if (in[i] != 1 && in[i] != -1) return -1; }
        else if (in[i] > FIELD_CLAMP || in[i] < -FIELD_CLAMP) return -1;
    }
    for (int64_t i = 0; i < o->N; ++i) { if (o->kind == 0) o->hb[i] = (int8_t)in[i]; else o->g[i] = in[i]; }
    return 0;
}
int oracle_get_permutation(void* p, int32_t* t2r) {
    Oracle* o = (Oracle*)p;
    for (int t = 0; t < o->n; ++t) t2r[t] = o->t2r[t];
    return 0;
}
int oracle_set_permutation(void* p, const int32_t* t2r) {
    Oracle* o = (Oracle*)p;
    std::vector<int32_t> r2t(o->R, -1);
    for (int t = 0; t < o->n; ++t) {
        if (t2r[t] < 0 || t2r[t] >= o->R || r2t[t2r[t]] != -1) return -1;
        r2t[t2r[t]] = t;
    }
    for (int t = 0; t < o->n; ++t) o->t2r[t] = t2r[t];
    o->r2t = r2t;
    return 0;
}
int oracle_get_temperatures(void* p, double* T, int* n) {
    Oracle* o = (Oracle*)p;
    if (n) *n = o->n;
    if (T) for (int t = 0; t < o->n; ++t) T[t] = o->T[t];
    return 0;
}
int oracle_get_counters(void* p, uint64_t* sweep_index, uint64_t* exchange_step) {
    Oracle* o = (Oracle*)p;
    if (sweep_index) *sweep_index = o->sweep_g;
    if (exchange_step) *exchange_step = o->xstep;
    return 0;
}
int oracle_set_counters(void* p, uint64_t sweep_index, uint64_t exchange_step) {
    Oracle* o = (Oracle*)p;
    o->sweep_g = sweep_index; o->xstep = exchange_step;
    return 0;
}
// current integer energy terms by temperature rank
int oracle_get_energy_terms(void* p, int64_t* Eb, int64_t* Ef, int64_t* Msum) {
    Oracle* o = (Oracle*)p;
    if (!o->have_T) return -2;
    for (int t = 0; t < o->n; ++t) {
        const Measurement m = o->measure_slot(o->t2r[t]);
        if (Eb) Eb[t] = m.Eb;
        if (Ef) Ef[t] = m.Ef;
        if (Msum) Msum[t] = m.Msum;
    }
    return 0;
}
int64_t oracle_timeseries_steps(void* p) { return ((Oracle*)p)->series_steps; }
// series laid out [step][rank] for the current n
int oracle_get_timeseries(void* p, int64_t* Eb, int64_t* Ef, int64_t* Msum) {
    Oracle* o = (Oracle*)p;
    const size_t m = o->series.size();
    for (size_t q = 0; q < m; ++q) {
        if (Eb) Eb[q] = o->series[q].Eb;
        if (Ef) Ef[q] = o->series[q].Ef;
        if (Msum) Msum[q] = o->series[q].Msum;
    }
    return 0;
}
int oracle_get_exchange_counts(void* p, uint64_t* att, uint64_t* acc) {
    Oracle* o = (Oracle*)p;
    for (int t = 0; t < o->n - 1; ++t) { if (att) att[t] = o->att[t]; if (acc) acc[t] = o->acc[t]; }
    return 0;
}
// threshold (0..2^32) the next attempt at site (x,y,z) of `slot` would be compared with
uint64_t oracle_site_threshold(void* p, int slot, int x, int y, int z) {
    return ((Oracle*)p)->site_threshold(slot, x, y, z);
}
// bimodal table entry thr[rank][k][b]
uint64_t oracle_bimodal_threshold(void* p, int rank, int k, int b) {
    Oracle* o = (Oracle*)p;
    if (o->kind != 0 || rank < 0 || rank >= o->n || k < 0 || k > 6 || b < 0 || b > 1) return ~0ull;
    return o->thr_bimodal[(size_t)rank * 14 + k * 2 + b];
}
double oracle_energy_from_terms(void* p, int64_t Eb, int64_t Ef) {
    Measurement m{Eb, Ef, 0};
    return ((Oracle*)p)->energy_of(m);
}
// Thermal moments of the measurement series (one measurement per parallel-tempering step), per temperature
// rank, over the steps [skip, steps): out[t][0..4] = <e>, <e^2>, <|m|>, <m^2>, <m^4> with e = E/N the energy per site
// ("E is the average energy per site") and m = (1/V) sum_i s_i (Eq. 11).  Plain running sums
// in step order.  The observables of Eq. 11-13 follow from these (oracle/__init__.py: thermal_observables).
int oracle_thermal_moments(void* p, int64_t skip, double* out) {
    Oracle* o = (Oracle*)p;
    const int64_t steps = o->series_steps;
    if (skip < 0 || skip >= steps || !out) return -1;
    const int n = o->n;
    const double cnt = (double)(steps - skip);
    for (int t = 0; t < n; ++t) {
        double se = 0, se2 = 0, sa = 0, sm2 = 0, sm4 = 0;
        for (int64_t q = skip; q < steps; ++q) {
            const Measurement& ms = o->series[(size_t)q * n + t];
            const double e = o->energy_of(ms) / (double)o->N;
            const double m = (double)ms.Msum / (double)o->N;
            se += e; se2 += e * e; sa += std::fabs(m); sm2 += m * m; sm4 += (m * m) * (m * m);
        }
        out[5 * t + 0] = se / cnt; out[5 * t + 1] = se2 / cnt; out[5 * t + 2] = sa / cnt;
        out[5 * t + 3] = sm2 / cnt; out[5 * t + 4] = sm4 / cnt;
    }
    return 0;
}
// run exactly one half-sweep / one exchange step (for invariants checked between them)
int oracle_half_sweep(void* p, int slot, int colour, uint64_t sweep_index) {
    Oracle* o = (Oracle*)p;
    if (!o->have_T || slot < 0 || slot >= o->R || o->r2t[slot] < 0) return -1;
    o->half_sweep(slot, colour, sweep_index);
    return 0;
}
int oracle_exchange_step(void* p) {
    Oracle* o = (Oracle*)p;
    if (!o->have_T) return -2;
    o->exchange_step();
    return 0;
}
const char* oracle_last_error(void* p) { return ((Oracle*)p)->err.c_str(); }

}  // extern "C"

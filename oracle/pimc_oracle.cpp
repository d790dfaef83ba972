// ORACLE -- TEST INFRASTRUCTURE ONLY.
//
// Plain, serial, fp64 C++17 restatement of the hot path of arXiv 1103.4887
// (Quinn & Abarbanel): Metropolis checkerboard sweeps over the discretised path
// X = {x_0..x_M} and sequential whole-path parameter moves, under the action
//     A(X,p) = sum_{n=1..M} (Rm/2) |y_n - h(x_n)|^2                       (Eq. A_o)
//            + sum_{n=0..M-1} sum_a (Rf_a/2) ((x_{n+1,a}-x_{n,a}) - g_a(x_n,p))^2   (A_d,
//              in the RK4-map form BASELINE.json's north_star names)
// It follows the algorithm step by step in the paper's order (Fig. 1
// steps (a)-(i); Eq. 9).  No blocking, fusion or reordering.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may build, load or call this file.  It shares NO code with the CUDA library under
// paper_1103_4887_b200/ (no headers, helpers, tables or constants) and the product never
// routes through it.  Build: g++ -O2 -std=c++17 -ffp-contract=off -shared -fPIC.
//
// Pins (tests/ -m "not gpu"): Philox vs the published known-answer vectors and vs cuRAND's
// host code path; RK4 order-4 convergence; local dA vs brute-force A(X')-A(X) in long
// double; antisymmetry, telescoping, cache coherence, order independence; the linear
// model's stationary distribution vs the closed-form Gaussian posterior (banded solve and
// Kalman/RTS); 1-site textbook Gaussian; the gate kinetics' widths one and half a width from the
// midpoint with Table 1's numbers typed from PAPER.md:288-294 (tests/test_oracle_model.py); the
// fp32-state branches against exact rational arithmetic (tests/test_oracle_fp32_state.py).  PARITY UNPINNED: the Hodgkin-Huxley posterior
// moments themselves (Table 2 needs the paper's data and 1e6 tuned
// iterations) -- for HH the chain is pinned only through its parts (model, dA, rule, RNG).
//
// Options beyond that default path, each following the passage it cites and pinned in its own test file:
//   set_discretisation(1)  the paper's trapezoid rule, Eq. 7             tests/test_oracle_trapezoid.py
//   set_update_mode(1)     one component per proposal, PAPER.md:226-230               tests/test_oracle_componentwise.py
//   model 2                classic Hodgkin-Huxley alpha/beta rate functions            tests/test_oracle_classic_hh.py
//   set_annealing          beta on the dynamics term, Eq. 10          tests/test_oracle_annealing.py
//   set_tuning             step-size adjustment rule, PAPER.md:224-230                 tests/test_oracle_tuning.py
//   param_trace            record of the parameters at every accumulated sweep, Fig. 4   tests/test_oracle_diagnostics.py
//   residuals / residual_stats   model and observation errors eps_n, delta_n, PAPER.md:331             tests/test_oracle_diagnostics.py
// oracle/count_work.py restates this file's arithmetic on a counting number type (validated bit for bit against it) to count
// the algorithmic work per unit that bench.py's roofline credits (tests/test_work_model.py).
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <new>
#include <string>
#include <vector>

namespace {

constexpr int MODEL_LINEAR = 0;
constexpr int MODEL_HH = 1;
constexpr int MODEL_HH_CLASSIC = 2;   // same V equation, the classic alpha/beta rate functions
constexpr int MAXD = 8;

// ---------------------------------------------------------------------------------------
// R1. Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): a 4-word counter and a 2-word key.
// One round: (hi0,lo0) = 0xD2511F53 * c0 ; (hi1,lo1) = 0xCD9E8D57 * c2 ;
//            c <- (hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0).  Between rounds the key is
// bumped by (0x9E3779B9, 0xBB67AE85).  Ten rounds.
// ---------------------------------------------------------------------------------------
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) {
            k0 += 0x9E3779B9u;
            k1 += 0xBB67AE85u;
        }
        const uint64_t prod0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        const uint64_t prod1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        const uint32_t hi0 = (uint32_t)(prod0 >> 32), lo0 = (uint32_t)prod0;
        const uint32_t hi1 = (uint32_t)(prod1 >> 32), lo1 = (uint32_t)prod1;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n1 = lo1;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        const uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// R2. counter = (c0 = site n or parameter l, c1 = sweep t low 32 bits, c2 = chain,
//                c3 = stream | block<<8 | (t>>32)<<16), key = (seed_lo, seed_hi).
enum { STREAM_STATE_PROPOSAL = 0, STREAM_STATE_ACCEPT = 1, STREAM_PARAM = 2 };

void draw_words(uint64_t seed, uint64_t t, uint32_t chain, uint32_t index, uint32_t stream,
                uint32_t block, uint32_t out[4]) {
    const uint32_t ctr[4] = {index, (uint32_t)(t & 0xFFFFFFFFull), chain,
                             stream | (block << 8) | ((uint32_t)(t >> 32) << 16)};
    const uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32)};
    philox4x32_10(ctr, key, out);
}

// R3. uniforms strictly inside (0,1), exactly representable.
double u01_from_word(uint32_t w) { return ((double)w + 0.5) * 0x1p-32; }                 // proposals
double u01_from_two_words(uint32_t w0, uint32_t w1) {                                    // accept test
    const uint64_t v = (((uint64_t)w1 << 32) | (uint64_t)w0) >> 12;                      // 52 bits
    return ((double)v + 0.5) * 0x1p-52;
}
float u01f_from_word(uint32_t w) { return ((float)(w >> 9) + 0.5f) * 0x1p-23f; }         // fp32-state mode

// R4. Box-Muller: z0 = sqrt(-2 ln u1) cos(2 pi u2), z1 = sqrt(-2 ln u1) sin(2 pi u2).
const double TWO_PI = 6.283185307179586476925286766559;
void box_muller(double u1, double u2, double* z0, double* z1) {
    const double r = std::sqrt(-2.0 * std::log(u1));
    const double a = TWO_PI * u2;
    *z0 = r * std::cos(a);
    *z1 = r * std::sin(a);
}

// ---------------------------------------------------------------------------------------
// S1. Models.
// HH (Eq. 11-14; parameter vector and state order per SURVEY.md §0 D4, D5):
//   x = (V, m, h, n), p = (gNa, gK, gL, ENa, EK, EL, C)
//   dV/dt = (I + gNa m^3 h (ENa - V) + gK n^4 (EK - V) + gL (EL - V)) / C
//   da/dt = (a_inf(V) - a) / tau_a(V),  a_inf = 1/2 + 1/2 tanh((V - V_a)/dV_a)          (Eq. 13)
//                                       tau_a = tau_a0 + tau_a1 (1 - tanh^2((V - V_a)/dV_a))   (Eq. 14)
//   Table 1 constants with V_a shifted by -65 mV.
// ---------------------------------------------------------------------------------------
struct Kinetics { double Va, dVa, tau0, tau1; };
const Kinetics KIN_M = {-40.0, 15.0, 0.1, 0.4};
const Kinetics KIN_H = {-60.0, -15.0, 1.0, 7.0};
const Kinetics KIN_N = {-55.0, 30.0, 1.0, 5.0};

double gate_rate(const Kinetics& k, double V, double a) {
    const double th = std::tanh((V - k.Va) / k.dVa);
    const double a_inf = 0.5 + 0.5 * th;
    const double tau = k.tau0 + k.tau1 * (1.0 - th * th);
    return (a_inf - a) / tau;
}

// Classic Hodgkin-Huxley rate functions (Hodgkin & Huxley 1952, voltages shifted so that rest is -65 mV; BASELINE.json
// config 0 says "standard HH"):  da/dt = alpha_a(V) (1 - a) - beta_a(V) a  with
//   alpha_m = 0.1 (V+40) / (1 - exp(-(V+40)/10))    beta_m = 4 exp(-(V+65)/18)
//   alpha_h = 0.07 exp(-(V+65)/20)                  beta_h = 1 / (1 + exp(-(V+35)/10))
//   alpha_n = 0.01 (V+55) / (1 - exp(-(V+55)/10))   beta_n = 0.125 exp(-(V+65)/80)
// u / (1 - exp(-u)) has a removable singularity at u = 0 (value 1); expm1 keeps it accurate nearby.
double u_over_1mexp(double u) { return u == 0.0 ? 1.0 : u / -std::expm1(-u); }

void classic_gate_rates(double V, double m, double h, double n, double* Fg) {
    const double am = u_over_1mexp((V + 40.0) / 10.0), bm = 4.0 * std::exp(-(V + 65.0) / 18.0);          // 0.1 * 10 * u/(1-e^-u)
    const double ah = 0.07 * std::exp(-(V + 65.0) / 20.0), bh = 1.0 / (1.0 + std::exp(-(V + 35.0) / 10.0));
    const double an = 0.1 * u_over_1mexp((V + 55.0) / 10.0), bn = 0.125 * std::exp(-(V + 65.0) / 80.0);  // 0.01 * 10 * u/(1-e^-u)
    Fg[0] = am * (1.0 - m) - bm * m;
    Fg[1] = ah * (1.0 - h) - bh * h;
    Fg[2] = an * (1.0 - n) - bn * n;
}

void hh_rhs(const double* x, const double* p, double I, double* F, int model = MODEL_HH) {
    const double V = x[0], m = x[1], h = x[2], n = x[3];
    const double gNa = p[0], gK = p[1], gL = p[2], ENa = p[3], EK = p[4], EL = p[5], C = p[6];
    F[0] = (I + gNa * (m * m * m) * h * (ENa - V) + gK * (n * n * n * n) * (EK - V) + gL * (EL - V)) / C;
    if (model == MODEL_HH_CLASSIC) { classic_gate_rates(V, m, h, n, F + 1); return; }
    F[1] = gate_rate(KIN_M, V, m);
    F[2] = gate_rate(KIN_H, V, h);
    F[3] = gate_rate(KIN_N, V, n);
}

// S2. One step.  HH: classical RK4 increment g = (dt/6)(k1 + 2 k2 + 2 k3 + k4) with the current
// at the midpoint taken as (I_n + I_{n+1})/2.  Linear: the map is
// f(x) = A x with A = p (row-major D*D), g = A x - x.  f = x + g in both cases.
void step_increment(int model, int D, const double* x, const double* p, double I0, double I1,
                    double dt, double* g) {
    if (model == MODEL_LINEAR) {
        for (int a = 0; a < D; ++a) {
            double f = 0.0;
            for (int b = 0; b < D; ++b) f += p[a * D + b] * x[b];
            g[a] = f - x[a];
        }
        return;
    }
    const double Ih = 0.5 * (I0 + I1);
    double k1[4], k2[4], k3[4], k4[4], xs[4];
    hh_rhs(x, p, I0, k1, model);
    for (int a = 0; a < 4; ++a) xs[a] = x[a] + 0.5 * dt * k1[a];
    hh_rhs(xs, p, Ih, k2, model);
    for (int a = 0; a < 4; ++a) xs[a] = x[a] + 0.5 * dt * k2[a];
    hh_rhs(xs, p, Ih, k3, model);
    for (int a = 0; a < 4; ++a) xs[a] = x[a] + dt * k3[a];
    hh_rhs(xs, p, I1, k4, model);
    for (int a = 0; a < 4; ++a) g[a] = (dt / 6.0) * (k1[a] + 2.0 * k2[a] + 2.0 * k3[a] + k4[a]);
}

int model_np(int model, int D) { return (model == MODEL_HH || model == MODEL_HH_CLASSIC) ? 7 : D * D; }

// Neumaier compensated accumulator (S4: parameter-move sum in index order).
struct Neumaier {
    double s = 0.0, c = 0.0;
    void add(double v) {
        const double t = s + v;
        if (std::fabs(s) >= std::fabs(v)) c += (s - t) + v; else c += (v - t) + s;
        s = t;
    }
    double value() const { return s + c; }
};

struct HistSel { int site, comp; double lo, hi, width; };

struct Chain {
    int model, D, L, M, Np, state_dtype;     // state_dtype 64 or 32 (state values rounded to float)
    double dt, Rm;
    double Rf[MAXD];                          // model-error weights IN EFFECT this sweep: beta * Rf0 (beta = 1 unless annealing)
    double Rf0[MAXD];                         // the weights given at creation
    double beta0 = 1.0; uint64_t n_cool = 0, t_anneal = 0;   // simulated annealing of the dynamics term (Eq. 10)
    std::vector<double> x, g, y, I, p, lo, hi, wx, wp;
    int proposal_kind = 0;                    // 0 gaussian, 1 uniform
    // step-size auto-tuning: one step size per path component (n, a) and per parameter, adjusted every
    // tune_skip-th iteration from the acceptance counts of the last tune_skip iterations
    std::vector<double> ws;                   // (M+1)*D step sizes in use (all rows = wx until tuned)
    std::vector<uint32_t> nacc_s, nacc_p;     // accepted changes since the last adjustment, per (n, a) and per parameter
    bool tune = false; uint64_t tune_skip = 1, t_tune = 0; double f_acc = 0.23, alpha = 0.02;
    int update_mode = 0;                      // 0 = joint D-vector proposal, one decision per site (Fig. 1); 1 = one component at a time, D decisions per site (NEXT-2)
    int disc = 0;                             // model-error discretisation: 0 = explicit RK4 map (north_star), 1 = trapezoid rule (Eq. 7)
    uint64_t t = 0;                           // absolute sweep index
    uint32_t chain_id = 0;
    bool have_data = false, have_path = false;
    // S5 accumulators
    bool accum = false; uint64_t n_skip = 1, t_enable = 0, n_samples = 0;
    std::vector<double> cx, cp, S1x, S2x, S1p, S2p;
    // optional record of the parameters at every accumulated sweep (Fig. 4: "the evolution of one of the parameters")
    bool ptrace_on = false; std::vector<double> ptrace;
    // optional running sums of the model errors eps_n and observation errors delta_n of the accumulated paths
    bool resid_on = false; std::vector<double> E1, E2, D1, D2;
    // A6 counters: accepted / proposed, per component class and per parameter
    std::vector<uint64_t> acc, prop;
    // histograms
    std::vector<HistSel> hsel; int nbins = 0; std::vector<uint64_t> hist;
    // trace of the last sweep
    std::vector<double> tr_dA, tr_S, tr_logu, tr_xprop, tr_dAp, tr_Sp, tr_logup, tr_pprop;
    std::vector<uint8_t> tr_acc, tr_accp;
    std::string err;
};

double I_at(const Chain& c, int n) { return c.I.empty() ? 0.0 : c.I[n]; }

// The model-error term between steps n and n+1 is (Rf_a/2) r_a^2 with
//   disc 0 (RK4 map, BASELINE north_star):   r = (x_{n+1} - x_n) - g_n,            g_n = RK4 increment at x_n      (n = 0..M-1)
//   disc 1 (trapezoid, Eq. 7):  r = (x_{n+1} - x_n) - c_n - c_{n+1},  c_n = (dt/2) F(x_n, p; I_n)     (n = 0..M)
// i.e. the paper's eps_{n+1} = x_{n+1} - x_n - (dt/2)[F(x_{n+1}) + F(x_n)].  The cache array `g` holds g_n or c_n
// (the paper caches F_n).  Linear model in trapezoid form: F(x) = (A x - x)/dt, so c = (A x - x)/2.
int cache_len(const Chain& c) { return c.disc == 1 ? c.M + 1 : c.M; }

void half_rhs(int model, int D, const double* x, const double* p, double I, double dt, double* out) {
    if (model == MODEL_LINEAR) {
        for (int a = 0; a < D; ++a) {
            double f = 0.0;
            for (int b = 0; b < D; ++b) f += p[a * D + b] * x[b];
            out[a] = 0.5 * (f - x[a]);
        }
        return;
    }
    double F[4];
    hh_rhs(x, p, I, F, model);
    for (int a = 0; a < 4; ++a) out[a] = 0.5 * dt * F[a];
}

// cache entry n of the chain's discretisation at state x (n <= M-1 for disc 0, n <= M for disc 1)
void cache_value(const Chain& c, int n, const double* x, const double* p, double* out) {
    if (c.disc == 1) half_rhs(c.model, c.D, x, p, I_at(c, n), c.dt, out);
    else step_increment(c.model, c.D, x, p, I_at(c, n), I_at(c, n + 1), c.dt, out);
}

void rebuild_cache(Chain& c) {
    for (int n = 0; n < cache_len(c); ++n) cache_value(c, n, &c.x[(size_t)n * c.D], c.p.data(), &c.g[(size_t)n * c.D]);
}

// Local change of the action if x_n is replaced by xp (Fig. 1 (c)-(g)).
// gp (out, D values, only when n <= M-1) = increment at the proposal.  S (out) = sum of |every squared term|.
double site_delta_A(const Chain& c, int n, const double* xp, double* gp, double* S_out) {
    const int D = c.D, M = c.M;
    const double* xn = &c.x[(size_t)n * D];
    double dA = 0.0, S = 0.0;
    if (c.disc == 1) {
        // Fig. 1 (b)-(f) as printed: F' = F(x'_n); eps'_n, eps_n (term n-1 -> n), eps'_{n+1}, eps_{n+1} (term n -> n+1), delta'_n, delta_n
        cache_value(c, n, xp, c.p.data(), gp);                         // c'_n = (dt/2) F(x'_n): needed at every n, n = M included
        const double* cn = &c.g[(size_t)n * D];
        if (n >= 1) {
            const double* xm = &c.x[(size_t)(n - 1) * D];
            const double* cm = &c.g[(size_t)(n - 1) * D];
            for (int a = 0; a < D; ++a) {
                const double r_new = ((xp[a] - xm[a]) - cm[a]) - gp[a];
                const double r_old = ((xn[a] - xm[a]) - cm[a]) - cn[a];
                const double t_new = 0.5 * c.Rf[a] * r_new * r_new, t_old = 0.5 * c.Rf[a] * r_old * r_old;
                dA += t_new - t_old; S += t_new + t_old;
            }
            for (int l = 0; l < c.L; ++l) {
                const double d_new = c.y[(size_t)n * c.L + l] - xp[l];
                const double d_old = c.y[(size_t)n * c.L + l] - xn[l];
                const double t_new = 0.5 * c.Rm * d_new * d_new, t_old = 0.5 * c.Rm * d_old * d_old;
                dA += t_new - t_old; S += t_new + t_old;
            }
        }
        if (n <= M - 1) {
            const double* xq = &c.x[(size_t)(n + 1) * D];
            const double* cq = &c.g[(size_t)(n + 1) * D];
            for (int a = 0; a < D; ++a) {
                const double r_new = ((xq[a] - xp[a]) - gp[a]) - cq[a];
                const double r_old = ((xq[a] - xn[a]) - cn[a]) - cq[a];
                const double t_new = 0.5 * c.Rf[a] * r_new * r_new, t_old = 0.5 * c.Rf[a] * r_old * r_old;
                dA += t_new - t_old; S += t_new + t_old;
            }
        }
        if (S_out) *S_out = S;
        return dA;
    }
    if (n >= 1) {
        const double* xm = &c.x[(size_t)(n - 1) * D];
        const double* gm = &c.g[(size_t)(n - 1) * D];
        for (int a = 0; a < D; ++a) {                                  // model-error term n-1 -> n
            const double r_new = (xp[a] - xm[a]) - gm[a];
            const double r_old = (xn[a] - xm[a]) - gm[a];
            const double t_new = 0.5 * c.Rf[a] * r_new * r_new, t_old = 0.5 * c.Rf[a] * r_old * r_old;
            dA += t_new - t_old; S += t_new + t_old;
        }
        for (int l = 0; l < c.L; ++l) {                                // measurement term n (n = 1..M)
            const double d_new = c.y[(size_t)n * c.L + l] - xp[l];
            const double d_old = c.y[(size_t)n * c.L + l] - xn[l];
            const double t_new = 0.5 * c.Rm * d_new * d_new, t_old = 0.5 * c.Rm * d_old * d_old;
            dA += t_new - t_old; S += t_new + t_old;
        }
    }
    if (n <= M - 1) {
        step_increment(c.model, D, xp, c.p.data(), I_at(c, n), I_at(c, n + 1), c.dt, gp);
        const double* xq = &c.x[(size_t)(n + 1) * D];
        const double* gn = &c.g[(size_t)n * D];
        for (int a = 0; a < D; ++a) {                                  // model-error term n -> n+1
            const double r_new = (xq[a] - xp[a]) - gp[a];
            const double r_old = (xq[a] - xn[a]) - gn[a];
            const double t_new = 0.5 * c.Rf[a] * r_new * r_new, t_old = 0.5 * c.Rf[a] * r_old * r_old;
            dA += t_new - t_old; S += t_new + t_old;
        }
    }
    if (S_out) *S_out = S;
    return dA;
}

// Fig. 1 (a): proposal for site n at sweep t.  Gaussian: D normals from Box-Muller pairs
// (components 4b, 4b+1 from words 0,1 of block b; 4b+2, 4b+3 from words 2,3).  Uniform:
// x' = x + w (2u - 1).  In fp32-state mode the proposal is formed in float arithmetic.
void propose_site(const Chain& c, uint64_t seed, int n, double* xp) {
    const int D = c.D;
    const double* xn = &c.x[(size_t)n * D];
    for (int b = 0; 4 * b < D; ++b) {
        uint32_t w[4];
        draw_words(seed, c.t, c.chain_id, (uint32_t)n, STREAM_STATE_PROPOSAL, (uint32_t)b, w);
        if (c.state_dtype == 32) {
            for (int j = 0; j < 4 && 4 * b + j < D; ++j) {
                const int a = 4 * b + j;
                if (c.proposal_kind == 1) {
                    const float u = u01f_from_word(w[j]);
                    const float step = (float)c.ws[(size_t)n * D + a] * (2.0f * u - 1.0f);
                    xp[a] = (double)((float)xn[a] + step);
                }
            }
            if (c.proposal_kind == 0) {
                for (int pair = 0; pair < 2; ++pair) {
                    const float u1 = u01f_from_word(w[2 * pair]), u2 = u01f_from_word(w[2 * pair + 1]);
                    const float r = std::sqrt(-2.0f * std::log(u1));
                    const float ang = (float)TWO_PI * u2;
                    const float z[2] = {r * std::cos(ang), r * std::sin(ang)};
                    for (int j = 0; j < 2; ++j) {
                        const int a = 4 * b + 2 * pair + j;
                        if (a < D) xp[a] = (double)((float)xn[a] + (float)c.ws[(size_t)n * D + a] * z[j]);
                    }
                }
            }
        } else if (c.proposal_kind == 1) {
            for (int j = 0; j < 4 && 4 * b + j < D; ++j) {
                const int a = 4 * b + j;
                xp[a] = xn[a] + c.ws[(size_t)n * D + a] * (2.0 * u01_from_word(w[j]) - 1.0);
            }
        } else {
            for (int pair = 0; pair < 2; ++pair) {
                double z[2];
                box_muller(u01_from_word(w[2 * pair]), u01_from_word(w[2 * pair + 1]), &z[0], &z[1]);
                for (int j = 0; j < 2; ++j) {
                    const int a = 4 * b + 2 * pair + j;
                    if (a < D) xp[a] = xn[a] + c.ws[(size_t)n * D + a] * z[j];
                }
            }
        }
    }
}

double accept_log_u_state(const Chain& c, uint64_t seed, int n, int block = 0) {
    uint32_t w[4];
    draw_words(seed, c.t, c.chain_id, (uint32_t)n, STREAM_STATE_ACCEPT, (uint32_t)block, w);
    if (c.state_dtype == 32) return (double)std::log(u01f_from_word(w[0]));
    return std::log(u01_from_two_words(w[0], w[1]));
}

// S3 for one site: Fig. 1 (a)-(i).
void update_site(Chain& c, uint64_t seed, int n) {
    const int D = c.D;
    double xp[MAXD], gp[MAXD], S;
    propose_site(c, seed, n, xp);
    if (c.update_mode == 1) {
        // Component-wise updates (PAPER.md:226-230 keeps step sizes and acceptance counters "per component of the path"):
        // component a of site n is proposed with the SAME draw as in the joint move (x'_a = x_a + w_a z_a; x_a is untouched
        // by the other components' decisions), judged on its own with the accept uniform of block a of the accept stream,
        // and the next component starts from the state and cache this decision leaves.  Trace entries are per (n, a).
        for (int a = 0; a < D; ++a) {
            double xa[MAXD];
            for (int b = 0; b < D; ++b) xa[b] = c.x[(size_t)n * D + b];
            xa[a] = xp[a];
            const double dA = site_delta_A(c, n, xa, gp, &S);
            const double logu = accept_log_u_state(c, seed, n, a);
            const bool accept = logu < -dA;
            const size_t k = (size_t)n * D + a;
            c.tr_dA[k] = dA; c.tr_S[k] = S; c.tr_logu[k] = logu; c.tr_acc[k] = accept ? 1 : 0;
            c.tr_xprop[k] = xp[a];
            c.prop[a] += 1;
            if (accept) {
                c.acc[a] += 1; c.nacc_s[k] += 1;
                c.x[k] = xp[a];
                if (n < cache_len(c)) for (int b = 0; b < D; ++b) c.g[(size_t)n * D + b] = gp[b];
            }
        }
        return;
    }
    const double dA = site_delta_A(c, n, xp, gp, &S);
    const double logu = accept_log_u_state(c, seed, n);
    const bool accept = logu < -dA;                 // G3: NaN / +inf reject, dA <= 0 always accepts
    c.tr_dA[n] = dA; c.tr_S[n] = S; c.tr_logu[n] = logu; c.tr_acc[n] = accept ? 1 : 0;
    for (int a = 0; a < D; ++a) c.tr_xprop[(size_t)n * D + a] = xp[a];
    for (int a = 0; a < D; ++a) { c.prop[a] += 1; if (accept) c.acc[a] += 1; }
    if (accept) {
        for (int a = 0; a < D; ++a) c.nacc_s[(size_t)n * D + a] += 1;     // a joint move changes every component of the site
        for (int a = 0; a < D; ++a) c.x[(size_t)n * D + a] = xp[a];
        if (n < cache_len(c)) for (int a = 0; a < D; ++a) c.g[(size_t)n * D + a] = gp[a];
    }
}

// S3 half-sweep over the sites of one parity; `order` only changes the visiting order
// (0 forward, 1 reverse, 2 a fixed shuffle) -- PAPER.md:207 says it must not matter.
void half_sweep(Chain& c, uint64_t seed, int parity, int order) {
    std::vector<int> sites;
    for (int n = parity; n <= c.M; n += 2) sites.push_back(n);
    if (order == 1) for (size_t i = 0, j = sites.size(); i + 1 < j; ++i) { --j; std::swap(sites[i], sites[j]); }
    if (order == 2) {
        uint64_t s = 0x9E3779B97F4A7C15ull ^ (uint64_t)parity;
        for (size_t i = sites.size(); i > 1; --i) {
            s = s * 6364136223846793005ull + 1442695040888963407ull;
            std::swap(sites[i - 1], sites[(size_t)((s >> 33) % i)]);
        }
    }
    for (int n : sites) update_site(c, seed, n);
}

// Change of the action when the parameter vector becomes pnew on the current path: every model-error term changes
// (PAPER.md:199, 209).  gnew receives the cache under pnew; the sum runs over the terms in index order (Neumaier).
double param_delta_sum(const Chain& c, const double* pnew, std::vector<double>& gnew, double* S_out) {
    const int D = c.D, M = c.M, nc = cache_len(c);
    gnew.resize((size_t)(M + 1) * D);          // always room for the longer (trapezoid) cache: the arrays are swapped on accept
    for (int n = 0; n < nc; ++n) cache_value(c, n, &c.x[(size_t)n * D], pnew, &gnew[(size_t)n * D]);
    Neumaier sum; double S = 0.0;
    for (int n = 0; n < M; ++n)
        for (int a = 0; a < D; ++a) {
            const double d = c.x[(size_t)(n + 1) * D + a] - c.x[(size_t)n * D + a];
            double r_new = d - gnew[(size_t)n * D + a];
            double r_old = d - c.g[(size_t)n * D + a];
            if (c.disc == 1) { r_new -= gnew[(size_t)(n + 1) * D + a]; r_old -= c.g[(size_t)(n + 1) * D + a]; }
            const double t_new = 0.5 * c.Rf[a] * r_new * r_new, t_old = 0.5 * c.Rf[a] * r_old * r_old;
            sum.add(t_new - t_old); S += t_new + t_old;
        }
    if (S_out) *S_out = S;
    return sum.value();
}

// S4. Sequential parameter moves (row A4).
void parameter_moves(Chain& c, uint64_t seed) {
    const int D = c.D;
    std::vector<double> gnew, pnew(c.Np);
    for (int l = 0; l < c.Np; ++l) {
        c.tr_dAp[l] = std::numeric_limits<double>::quiet_NaN(); c.tr_Sp[l] = 0.0;
        c.tr_logup[l] = 0.0; c.tr_accp[l] = 0; c.tr_pprop[l] = c.p[l];
        if (!(c.wp[l] > 0.0)) continue;                                // frozen parameter
        uint32_t w[4];
        draw_words(seed, c.t, c.chain_id, (uint32_t)l, STREAM_PARAM, 0, w);
        double z0, z1, step;
        if (c.proposal_kind == 1) step = c.wp[l] * (2.0 * u01_from_word(w[0]) - 1.0);
        else { box_muller(u01_from_word(w[0]), u01_from_word(w[1]), &z0, &z1); step = c.wp[l] * z0; }
        double pl = c.p[l] + step;
        if (c.state_dtype == 32) pl = (double)((float)c.p[l] + (float)step);
        const double logu = std::log(u01_from_two_words(w[2], w[3]));
        c.tr_pprop[l] = pl; c.tr_logup[l] = logu;
        c.prop[D + l] += 1;
        if (!(pl >= c.lo[l] && pl <= c.hi[l])) continue;               // outside bounds => rejected
        pnew = c.p; pnew[l] = pl;
        double S = 0.0;
        const double dA = param_delta_sum(c, pnew.data(), gnew, &S);
        const bool accept = logu < -dA;
        c.tr_dAp[l] = dA; c.tr_Sp[l] = S; c.tr_accp[l] = accept ? 1 : 0;
        if (accept) { c.p[l] = pl; c.g.swap(gnew); c.acc[D + l] += 1; c.nacc_p[l] += 1; }
    }
}

// Model errors and observation errors of the current path ("look at the model errors, eps_n, and the observation
// errors, delta_n ... functions of the path"), in the discretisation in use:
//   eps_{n,a}   = (x_{n+1,a} - x_{n,a}) - g_{n,a}                      n = 0..M-1   (RK4 map; trapezoid: ... - c_n - c_{n+1})
//   delta_{n,l} = y_{n,l} - x_{n,l}                                     n = 1..M     (delta_0 = 0: y_0 is not in the action)
// so that A(X) = sum (Rm/2) delta^2 + sum (Rf_a/2) eps^2 exactly as the action is defined (pinned that way in the tests).
void residuals(const Chain& c, double* eps /* M*D */, double* delta /* (M+1)*L */) {
    const int D = c.D, M = c.M, L = c.L;
    for (int n = 0; n < M; ++n)
        for (int a = 0; a < D; ++a) {
            double r = (c.x[(size_t)(n + 1) * D + a] - c.x[(size_t)n * D + a]) - c.g[(size_t)n * D + a];
            if (c.disc == 1) r -= c.g[(size_t)(n + 1) * D + a];
            eps[(size_t)n * D + a] = r;
        }
    for (int n = 0; n <= M; ++n)
        for (int l = 0; l < L; ++l) delta[(size_t)n * L + l] = n >= 1 ? c.y[(size_t)n * L + l] - c.x[(size_t)n * D + l] : 0.0;
}
void accumulate_residuals(Chain& c) {
    std::vector<double> eps((size_t)c.M * c.D), del((size_t)(c.M + 1) * c.L);
    residuals(c, eps.data(), del.data());
    for (size_t i = 0; i < eps.size(); ++i) { c.E1[i] += eps[i]; c.E2[i] += eps[i] * eps[i]; }
    for (size_t i = 0; i < del.size(); ++i) { c.D1[i] += del[i]; c.D2[i] += del[i] * del[i]; }
}

// S5. Running moments about the reference point c (values at the last reset) + histograms.
void accumulate(Chain& c) {
    const size_t nx = (size_t)(c.M + 1) * c.D;
    for (size_t i = 0; i < nx; ++i) { const double d = c.x[i] - c.cx[i]; c.S1x[i] += d; c.S2x[i] += d * d; }
    for (int l = 0; l < c.Np; ++l) { const double d = c.p[l] - c.cp[l]; c.S1p[l] += d; c.S2p[l] += d * d; }
    for (size_t s = 0; s < c.hsel.size(); ++s) {
        const HistSel& h = c.hsel[s];
        const double v = h.site < 0 ? c.p[h.comp] : c.x[(size_t)h.site * c.D + h.comp];
        uint64_t* bins = &c.hist[s * (size_t)(c.nbins + 2)];
        if (!(v >= h.lo)) bins[0] += 1;                               // underflow (and NaN)
        else if (v >= h.hi) bins[c.nbins + 1] += 1;                   // overflow
        else {
            long long b = (long long)std::floor((v - h.lo) / h.width);
            if (b >= c.nbins) b = c.nbins - 1;
            bins[1 + b] += 1;
        }
    }
    if (c.ptrace_on) c.ptrace.insert(c.ptrace.end(), c.p.begin(), c.p.end());
    if (c.resid_on) accumulate_residuals(c);
    c.n_samples += 1;
}

void reset_moments(Chain& c) {
    c.ptrace.clear();
    std::fill(c.E1.begin(), c.E1.end(), 0.0); std::fill(c.E2.begin(), c.E2.end(), 0.0);
    std::fill(c.D1.begin(), c.D1.end(), 0.0); std::fill(c.D2.begin(), c.D2.end(), 0.0);
    c.cx = c.x; c.cp = c.p;
    std::fill(c.S1x.begin(), c.S1x.end(), 0.0); std::fill(c.S2x.begin(), c.S2x.end(), 0.0);
    std::fill(c.S1p.begin(), c.S1p.end(), 0.0); std::fill(c.S2p.begin(), c.S2p.end(), 0.0);
    std::fill(c.hist.begin(), c.hist.end(), 0ull);
    c.n_samples = 0; c.t_enable = c.t;
}

// Step-size adjustment: Delta_i <- Delta_i [1 + alpha (N_acc,i / N_skip - f_acc)] for every path component
// and every parameter, every N_skip-th iteration while tuning is on; N_acc,i restarts from zero.
void maybe_tune(Chain& c) {
    if (!c.tune) return;
    const uint64_t k = c.t - c.t_tune + 1;               // iterations completed since tuning was switched on
    if (k % c.tune_skip != 0) return;
    const double ns = (double)c.tune_skip;
    for (size_t i = 0; i < c.ws.size(); ++i) {
        c.ws[i] = c.ws[i] * (1.0 + c.alpha * ((double)c.nacc_s[i] / ns - c.f_acc));
        c.nacc_s[i] = 0;
    }
    for (int l = 0; l < c.Np; ++l) {
        c.wp[l] = c.wp[l] * (1.0 + c.alpha * ((double)c.nacc_p[l] / ns - c.f_acc));
        c.nacc_p[l] = 0;
    }
}

// Simulated annealing: the dynamics term A_d carries a multiplier beta that starts at beta0 < 1 and is
// multiplied by f_beta = (1/beta0)^(1/N_cool) (Eq. 10) after each iteration until it reaches 1; the observation term does
// not.  After k iterations beta = beta0 f_beta^k = beta0^(1 - k/N_cool), evaluated in that closed form.
double annealing_beta(const Chain& c) {
    if (c.n_cool == 0 || c.t < c.t_anneal) return 1.0;
    const uint64_t k = c.t - c.t_anneal;
    if (k >= c.n_cool) return 1.0;
    return std::exp(std::log(c.beta0) * (1.0 - (double)k / (double)c.n_cool));
}
void apply_annealing(Chain& c) {
    const double beta = annealing_beta(c);
    for (int a = 0; a < c.D; ++a) c.Rf[a] = beta * c.Rf0[a];
}

// Test-only "truth": the full action in long double, straight from the definition.
long double full_action(const Chain& c, const double* x, const double* p) {
    const int D = c.D;
    long double A = 0.0L;
    for (int n = 1; n <= c.M; ++n)
        for (int l = 0; l < c.L; ++l) {
            const long double d = (long double)c.y[(size_t)n * c.L + l] - (long double)x[(size_t)n * D + l];
            A += 0.5L * (long double)c.Rm * d * d;
        }
    double g[MAXD], g1[MAXD];
    for (int n = 0; n < c.M; ++n) {
        cache_value(c, n, &x[(size_t)n * D], p, g);
        if (c.disc == 1) cache_value(c, n + 1, &x[(size_t)(n + 1) * D], p, g1);
        for (int a = 0; a < D; ++a) {
            long double r = ((long double)x[(size_t)(n + 1) * D + a] - (long double)x[(size_t)n * D + a]) - (long double)g[a];
            if (c.disc == 1) r -= (long double)g1[a];
            A += 0.5L * (long double)c.Rf[a] * r * r;
        }
    }
    return A;
}

}  // namespace

// =========================================================================================
// C interface for ctypes (tests and bench only).
// =========================================================================================
extern "C" {

void orc_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }
void orc_draw_words(uint64_t seed, uint64_t t, uint32_t chain, uint32_t index, uint32_t stream, uint32_t block,
                    uint32_t* out) { draw_words(seed, t, chain, index, stream, block, out); }
// n counters (n,4) with one key -> n outputs (n,4); for the RNG-quality tests.
void orc_philox_bulk(uint64_t n, const uint32_t* ctrs, const uint32_t* key, uint32_t* out) {
    for (uint64_t i = 0; i < n; ++i) philox4x32_10(ctrs + 4 * i, key, out + 4 * i);
}
double orc_u01_from_word(uint32_t w) { return u01_from_word(w); }
double orc_u01_from_two_words(uint32_t w0, uint32_t w1) { return u01_from_two_words(w0, w1); }
float orc_u01f_from_word(uint32_t w) { return u01f_from_word(w); }
void orc_box_muller(double u1, double u2, double* z) { box_muller(u1, u2, &z[0], &z[1]); }
int orc_model_np(int model, int D) { return model_np(model, D); }
void orc_rhs(int model, const double* x, const double* p, double I, double* F) { if (model == MODEL_HH || model == MODEL_HH_CLASSIC) hh_rhs(x, p, I, F, model); }
void orc_step_increment(int model, int D, const double* x, const double* p, double I0, double I1, double dt,
                        double* g) { step_increment(model, D, x, p, I0, I1, dt, g); }

void* orc_create(int model, int D, int L, int M, double dt, double Rm, const double* Rf, const double* p0,
                 int state_dtype, uint32_t chain_id) {
    if (!(model == MODEL_LINEAR || model == MODEL_HH || model == MODEL_HH_CLASSIC)) return nullptr;
    if (model != MODEL_LINEAR && D != 4) return nullptr;
    if (D < 1 || D > MAXD || (model == MODEL_LINEAR && D > 4) || L < 0 || L > D || M < 1) return nullptr;
    if (!(state_dtype == 64 || state_dtype == 32)) return nullptr;
    Chain* c = new (std::nothrow) Chain();
    if (!c) return nullptr;
    c->model = model; c->D = D; c->L = L; c->M = M; c->Np = model_np(model, D); c->state_dtype = state_dtype;
    c->dt = dt; c->Rm = Rm; c->chain_id = chain_id;
    for (int a = 0; a < D; ++a) c->Rf[a] = c->Rf0[a] = Rf[a];
    const size_t nx = (size_t)(M + 1) * D;
    c->x.assign(nx, 0.0); c->g.assign((size_t)(M + 1) * D, 0.0); c->y.assign((size_t)(M + 1) * (L > 0 ? L : 1), 0.0);
    c->p.assign(p0, p0 + c->Np);
    if (state_dtype == 32) for (double& v : c->p) v = (double)(float)v;
    c->lo.assign(c->Np, -std::numeric_limits<double>::infinity());
    c->hi.assign(c->Np, std::numeric_limits<double>::infinity());
    c->wx.assign(D, 0.0); c->wp.assign(c->Np, 0.0);
    c->ws.assign(nx, 0.0); c->nacc_s.assign(nx, 0); c->nacc_p.assign(c->Np, 0);
    c->cx.assign(nx, 0.0); c->S1x.assign(nx, 0.0); c->S2x.assign(nx, 0.0);
    c->cp.assign(c->Np, 0.0); c->S1p.assign(c->Np, 0.0); c->S2p.assign(c->Np, 0.0);
    c->acc.assign(D + c->Np, 0); c->prop.assign(D + c->Np, 0);
    c->tr_dA.assign(nx, 0.0); c->tr_S.assign(nx, 0.0); c->tr_logu.assign(nx, 0.0);     // (M+1) entries used by joint updates, (M+1) D by component-wise ones
    c->tr_xprop.assign(nx, 0.0); c->tr_acc.assign(nx, 0);
    c->tr_dAp.assign(c->Np, 0.0); c->tr_Sp.assign(c->Np, 0.0); c->tr_logup.assign(c->Np, 0.0);
    c->tr_pprop.assign(c->Np, 0.0); c->tr_accp.assign(c->Np, 0);
    return c;
}
void orc_destroy(void* h) { delete (Chain*)h; }

void orc_set_data(void* h, const double* y, const double* I) {
    Chain& c = *(Chain*)h;
    if (c.L > 0) c.y.assign(y, y + (size_t)(c.M + 1) * c.L);
    if (I) c.I.assign(I, I + (c.M + 1)); else c.I.clear();
    if (c.state_dtype == 32) { for (double& v : c.y) v = (double)(float)v; for (double& v : c.I) v = (double)(float)v; }
    c.have_data = true;
    if (c.have_path) rebuild_cache(c);
}
void orc_set_path(void* h, const double* x) {
    Chain& c = *(Chain*)h;
    c.x.assign(x, x + (size_t)(c.M + 1) * c.D);
    if (c.state_dtype == 32) for (double& v : c.x) v = (double)(float)v;
    c.have_path = true;
    rebuild_cache(c);
}
void orc_set_params(void* h, const double* p) {
    Chain& c = *(Chain*)h;
    c.p.assign(p, p + c.Np);
    if (c.state_dtype == 32) for (double& v : c.p) v = (double)(float)v;
    if (c.have_path) rebuild_cache(c);
}
void orc_get_path(void* h, double* x, double* p) {
    Chain& c = *(Chain*)h;
    if (x) std::memcpy(x, c.x.data(), c.x.size() * sizeof(double));
    if (p) std::memcpy(p, c.p.data(), c.p.size() * sizeof(double));
}
// cache entries in use: M (RK4 map) or M+1 (trapezoid) rows of D values
int orc_cache_len(void* h) { return cache_len(*(Chain*)h); }
void orc_get_cache(void* h, double* g) { Chain& c = *(Chain*)h; std::memcpy(g, c.g.data(), (size_t)cache_len(c) * c.D * sizeof(double)); }
// 0 = explicit RK4 map (default), 1 = trapezoid rule of the paper (Eq. 7)
int orc_set_discretisation(void* h, int disc) {
    Chain& c = *(Chain*)h;
    if (!(disc == 0 || disc == 1)) return -1;
    c.disc = disc;
    if (c.have_path) rebuild_cache(c);
    return 0;
}
// Start annealing at the current sweep index: beta0 in (0, 1], n_cool iterations (0 switches it off)
int orc_set_annealing(void* h, double beta0, uint64_t n_cool) {
    Chain& c = *(Chain*)h;
    if (!(beta0 > 0.0 && beta0 <= 1.0)) return -1;
    c.beta0 = beta0; c.n_cool = n_cool; c.t_anneal = c.t;
    apply_annealing(c);
    return 0;
}
double orc_annealing_beta(void* h) { return annealing_beta(*(Chain*)h); }
// 0 = joint proposal per site (default), 1 = component-wise
int orc_set_update_mode(void* h, int mode) {
    Chain& c = *(Chain*)h;
    if (!(mode == 0 || mode == 1)) return -1;
    c.update_mode = mode;
    return 0;
}
void orc_half_rhs(int model, int D, const double* x, const double* p, double I, double dt, double* out) { half_rhs(model, D, x, p, I, dt, out); }
void orc_set_proposal(void* h, const double* w_state, const double* w_param, int kind) {
    Chain& c = *(Chain*)h;
    c.wx.assign(w_state, w_state + c.D);
    if (w_param) c.wp.assign(w_param, w_param + c.Np); else c.wp.assign(c.Np, 0.0);
    c.proposal_kind = kind;
    c.ws.resize((size_t)(c.M + 1) * c.D);
    for (int n = 0; n <= c.M; ++n) for (int a = 0; a < c.D; ++a) c.ws[(size_t)n * c.D + a] = c.wx[a];
    c.nacc_s.assign(c.ws.size(), 0); c.nacc_p.assign(c.Np, 0);
}
// Step-size auto-tuning from the current sweep index on; enabled = 0 freezes the step sizes as they are.
int orc_set_tuning(void* h, int enabled, uint64_t n_skip, double f_acc, double alpha) {
    Chain& c = *(Chain*)h;
    if (enabled && (n_skip < 1 || !(f_acc > 0.0 && f_acc < 1.0) || !(alpha >= 0.0 && alpha < 1.0))) return -1;
    c.tune = enabled != 0;
    if (enabled) {
        c.tune_skip = n_skip; c.f_acc = f_acc; c.alpha = alpha; c.t_tune = c.t;
        std::fill(c.nacc_s.begin(), c.nacc_s.end(), 0u); std::fill(c.nacc_p.begin(), c.nacc_p.end(), 0u);
    }
    return 0;
}
void orc_get_widths(void* h, double* ws, double* wp) {
    Chain& c = *(Chain*)h;
    if (ws) std::memcpy(ws, c.ws.data(), c.ws.size() * 8);
    if (wp) std::memcpy(wp, c.wp.data(), c.wp.size() * 8);
}
void orc_set_bounds(void* h, const double* lo, const double* hi) {
    Chain& c = *(Chain*)h; c.lo.assign(lo, lo + c.Np); c.hi.assign(hi, hi + c.Np);
}
void orc_set_accum(void* h, int enabled, uint64_t n_skip) {
    Chain& c = *(Chain*)h;
    if (enabled && !c.accum) c.t_enable = c.t;
    c.accum = enabled != 0; c.n_skip = n_skip ? n_skip : 1;
}
void orc_reset_moments(void* h) { reset_moments(*(Chain*)h); }
uint64_t orc_sweep_index(void* h) { return ((Chain*)h)->t; }
void orc_set_sweep_index(void* h, uint64_t t) { ((Chain*)h)->t = t; apply_annealing(*(Chain*)h); }

int orc_hist_config(void* h, int n_sel, const int* site, const int* comp, const double* lo, const double* hi, int nbins) {
    Chain& c = *(Chain*)h;
    c.hsel.clear(); c.nbins = nbins;
    for (int s = 0; s < n_sel; ++s) c.hsel.push_back({site[s], comp[s], lo[s], hi[s], (hi[s] - lo[s]) / nbins});
    c.hist.assign((size_t)n_sel * (nbins + 2), 0ull);
    return 0;
}
void orc_hist(void* h, uint64_t* out) { Chain& c = *(Chain*)h; std::memcpy(out, c.hist.data(), c.hist.size() * sizeof(uint64_t)); }

// The iteration of PAPER.md:185-211: even half-sweep, odd half-sweep, parameters in sequence,
// statistics, t++.  `order` permutes sites within a half-sweep (testing PAPER.md:207).
// `do_params` = 0 skips S4 (used by tests of the state update alone).
int orc_sweep(void* h, uint64_t n_sweeps, uint64_t seed, int order, int do_params) {
    Chain& c = *(Chain*)h;
    if (!c.have_data || !c.have_path) return -2;
    for (uint64_t s = 0; s < n_sweeps; ++s) {
        apply_annealing(c);
        half_sweep(c, seed, 0, order);
        half_sweep(c, seed, 1, order);
        if (do_params) parameter_moves(c, seed);
        if (c.accum && ((c.t - c.t_enable) % c.n_skip) == 0) accumulate(c);
        maybe_tune(c);
        c.t += 1;
    }
    apply_annealing(c);          // the weights in effect always belong to the current sweep index
    return 0;
}

// S6 outputs: out = mean,var of x as (2, M+1, D), then mean,var of p as (2, Np).  Population variance.
// Record the parameters at every accumulated sweep from now on (cleared by orc_reset_moments).
void orc_param_trace_enable(void* h, int on) { Chain& c = *(Chain*)h; c.ptrace_on = on != 0; if (!on) c.ptrace.clear(); }
// out: (n_records, Np); returns the number of records held.
uint64_t orc_param_trace(void* h, double* out, uint64_t max_records) {
    Chain& c = *(Chain*)h;
    const uint64_t n = c.Np ? c.ptrace.size() / c.Np : 0, k = n < max_records ? n : max_records;
    if (out) std::memcpy(out, c.ptrace.data(), k * c.Np * sizeof(double));
    return n;
}
// eps (M, D), delta (M+1, L) of the current path
void orc_residuals(void* h, double* eps, double* delta) { residuals(*(Chain*)h, eps, delta); }
// Running means and variances of eps and delta over the accumulated sweeps (population form, like the moments)
void orc_residual_stats_enable(void* h, int on) {
    Chain& c = *(Chain*)h; c.resid_on = on != 0;
    c.E1.assign((size_t)c.M * c.D, 0.0); c.E2 = c.E1; c.D1.assign((size_t)(c.M + 1) * c.L, 0.0); c.D2 = c.D1;
}
// out: mean eps (M, D), var eps (M, D), mean delta (M+1, L), var delta (M+1, L)
uint64_t orc_residual_stats(void* h, double* out) {
    Chain& c = *(Chain*)h;
    const size_t ne = (size_t)c.M * c.D, nd = (size_t)(c.M + 1) * c.L;
    const double N = (double)c.n_samples;
    for (size_t i = 0; i < ne; ++i) { const double m = c.n_samples ? c.E1[i] / N : 0.0; out[i] = m; out[ne + i] = c.n_samples ? c.E2[i] / N - m * m : 0.0; }
    for (size_t i = 0; i < nd; ++i) { const double m = c.n_samples ? c.D1[i] / N : 0.0; out[2 * ne + i] = m; out[2 * ne + nd + i] = c.n_samples ? c.D2[i] / N - m * m : 0.0; }
    return c.n_samples;
}

uint64_t orc_moments(void* h, double* out) {
    Chain& c = *(Chain*)h;
    const size_t nx = (size_t)(c.M + 1) * c.D;
    const double N = (double)c.n_samples;
    for (size_t i = 0; i < nx; ++i) {
        const double m1 = c.n_samples ? c.S1x[i] / N : 0.0;
        out[i] = c.cx[i] + m1;
        out[nx + i] = c.n_samples ? c.S2x[i] / N - m1 * m1 : 0.0;
    }
    for (int l = 0; l < c.Np; ++l) {
        const double m1 = c.n_samples ? c.S1p[l] / N : 0.0;
        out[2 * nx + l] = c.cp[l] + m1;
        out[2 * nx + c.Np + l] = c.n_samples ? c.S2p[l] / N - m1 * m1 : 0.0;
    }
    return c.n_samples;
}
void orc_stats(void* h, uint64_t* out) {      // (2, D+Np): accepted, proposed
    Chain& c = *(Chain*)h; const int n = c.D + c.Np;
    for (int i = 0; i < n; ++i) { out[i] = c.acc[i]; out[n + i] = c.prop[i]; }
}
void orc_trace(void* h, double* dA, double* S, double* logu, uint8_t* acc, double* xprop, double* dAp, double* Sp,
               double* logup, uint8_t* accp, double* pprop) {
    Chain& c = *(Chain*)h;
    const size_t nt = (size_t)(c.M + 1) * (c.update_mode == 1 ? c.D : 1);      // per site, or per (site, component)
    if (dA) std::memcpy(dA, c.tr_dA.data(), nt * 8);
    if (S) std::memcpy(S, c.tr_S.data(), nt * 8);
    if (logu) std::memcpy(logu, c.tr_logu.data(), nt * 8);
    if (acc) std::memcpy(acc, c.tr_acc.data(), nt);
    if (xprop) std::memcpy(xprop, c.tr_xprop.data(), c.tr_xprop.size() * 8);
    if (dAp) std::memcpy(dAp, c.tr_dAp.data(), c.tr_dAp.size() * 8);
    if (Sp) std::memcpy(Sp, c.tr_Sp.data(), c.tr_Sp.size() * 8);
    if (logup) std::memcpy(logup, c.tr_logup.data(), c.tr_logup.size() * 8);
    if (accp) std::memcpy(accp, c.tr_accp.data(), c.tr_accp.size());
    if (pprop) std::memcpy(pprop, c.tr_pprop.data(), c.tr_pprop.size() * 8);
}

// Local dA of replacing x_n by xp on the CURRENT path (no RNG, no state change).
double orc_site_delta_A(void* h, int n, const double* xp, double* S) {
    Chain& c = *(Chain*)h; double gp[MAXD];
    return site_delta_A(c, n, xp, gp, S);
}
// Parameter-move dA of replacing p_l by pl on the current path (no RNG, no state change).
double orc_param_delta_A(void* h, int l, double pl, double* S_out) {
    Chain& c = *(Chain*)h;
    std::vector<double> pnew = c.p, gnew; pnew[l] = pl;
    return param_delta_sum(c, pnew.data(), gnew, S_out);
}
// Full action of an arbitrary (x, p) with this chain's data, accumulated in long double; returned as
// hi + lo doubles so ctypes callers keep the extra bits.
void orc_full_action(void* h, const double* x, const double* p, double* hi, double* lo) {
    Chain& c = *(Chain*)h;
    const long double A = full_action(c, x ? x : c.x.data(), p ? p : c.p.data());
    *hi = (double)A; *lo = (double)(A - (long double)*hi);
}

}  // extern "C"

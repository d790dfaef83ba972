// Model step increments g(x, p; I_n, I_{n+1}) for the PIMC kernels (row A0 of SURVEY.md §8(a)).
//   HH     : tanh-kinetics Hodgkin-Huxley neuron, PAPER.md:256-270 (Eq. 11-14), Table 1
//            shifted by -65 mV; one classical RK4 step of size dt, current at the half step = mean of the ends.
//   LINEAR : x -> A x with A = p (row-major D x D); g = A x - x.
// The caches hold the INCREMENT g, not f = x + g: the residual (x_{n+1} - x_n) - g_n then loses no bits to the
// +-65 mV offset of V (matters in fp32).
#pragma once
#include "pimc_math.cuh"

namespace pimc {

// ---------------------------------------------------------------------------------------------------
// KIN selects the gate kinetics: 0 = the paper's tanh forms, 1 = the classic alpha/beta rate functions
// (Hodgkin & Huxley 1952, rest at -65 mV; include/pimc.h PIMC_MODEL_HH_CLASSIC).  Everything else is shared.
template <typename R, int KIN> struct HHModelK {
    static constexpr int D = 4;
    static constexpr int NP = 7;
    static constexpr bool kTileMc = true;          // the many-chain tile-resident engine is compiled for this family

    // The parameter vector lives in shared memory (one copy per CTA); p[] = (gNa, gK, gL, ENa, EK, EL, C).
    // d a / dt = (a_inf(V) - a) / tau_a(V);  a_inf = 1/2 + 1/2 tanh(s), tau = tau0 + tau1 (1 - tanh^2 s), s = (V - Va)/dVa
    // Gate rates in one-exponential form.  With e = exp(2 s), q = e + 1:
    //   tanh s = (e-1)/q, a_inf = e/q, 1 - tanh^2 s = 4 e / q^2  =>  (a_inf - a)/tau = (e - a q) q / (tau0 q^2 + 4 tau1 e),
    //   and tau0 q^2 + 4 tau1 e = tau0 + e (2 tau0 + 4 tau1 + tau0 e) (two FMAs straight from e): one exponential and one
    //   reciprocal per gate instead of a tanh and a divide (gates_shared_exp below then shares the exponential between the gates).
    // dV/dt (Eq. 11 with the config's physical parameters): the only place the parameters enter
    static __device__ __forceinline__ R rhs_V(const R x[4], const R* __restrict__ p, R inv_C, R I) {
        const R V = x[0], m = x[1], h = x[2], n = x[3];
        const R n2 = n * n;
        const R cur = I + p[0] * (m * m * m) * h * (p[3] - V) + p[1] * (n2 * n2) * (p[4] - V) + p[2] * (p[5] - V);
        return cur * inv_C;
    }
    // d(m,h,n)/dt (Eq. 12-14): functions of the state only, not of the parameters
    static __device__ __forceinline__ void rhs_gates(const R x[4], R Fg[3]) {
        const R V = x[0], m = x[1], h = x[2], n = x[3];
        if constexpr (KIN == 1) {
            // da/dt = alpha_a (1 - a) - beta_a a; exponent arguments clamped so that nothing overflows inside the domain guard
            if constexpr (sizeof(R) == 8) {
                const double Vc = fmin(fmax(V, -6000.0), 6000.0);
                const double am = u_over_1mexp((Vc + 40.0) * 0.1), bm = 4.0 * exp_fast((Vc + 65.0) * (-1.0 / 18.0));
                const double ah = 0.07 * exp_fast((Vc + 65.0) * (-1.0 / 20.0)), bh = div_fast(1.0, 1.0 + exp_fast((Vc + 35.0) * -0.1));
                const double an = 0.1 * u_over_1mexp((Vc + 55.0) * 0.1), bn = 0.125 * exp_fast((Vc + 65.0) * (-1.0 / 80.0));
                Fg[0] = am * (1.0 - m) - bm * m;
                Fg[1] = ah * (1.0 - h) - bh * h;
                Fg[2] = an * (1.0 - n) - bn * n;
            } else {
                const float Vc = fminf(fmaxf(V, -700.0f), 700.0f);
                const float um = (Vc + 40.0f) * 0.1f, un = (Vc + 55.0f) * 0.1f;
                const float am = um == 0.0f ? 1.0f : um / -expm1f(-um), bm = 4.0f * expf(-(Vc + 65.0f) / 18.0f);
                const float ah = 0.07f * expf(-(Vc + 65.0f) / 20.0f), bh = 1.0f / (1.0f + expf(-(Vc + 35.0f) * 0.1f));
                const float an = un == 0.0f ? 0.1f : 0.1f * (un / -expm1f(-un)), bn = 0.125f * expf(-(Vc + 65.0f) / 80.0f);
                Fg[0] = am * (1.0f - m) - bm * m;
                Fg[1] = ah * (1.0f - h) - bh * h;
                Fg[2] = an * (1.0f - n) - bn * n;
            }
        } else if constexpr (sizeof(R) == 8) gates_shared_exp(V, m, h, n, Fg);
        else gates_shared_exp_f(V, m, h, n, Fg);
    }
    // ONE exponential for the three gates.  Table 1's widths are 15, -15 and 30 mV, so the three arguments
    // 2 s_a = 2 (V - V_a)/dV_a are (2V + 80)/15, -(2V + 120)/15 and (V + 55)/15: with u = exp((V + 55)/15) and w = u^2,
    //   e_n = u,   e_m = e^{-2} w,   e_h = e^{-2/3} / w.
    // m and n use the one-exponential form of gate_fast directly.  For h, numerator and denominator of
    // (e - a q) q / (tau0 + e (2 tau0 + 4 tau1 + tau0 e)) are multiplied by w^2:  with c = e^{-2/3}, Q = c + w,
    //   (c - a Q) Q / (tau0 w^2 + c (2 tau0 + 4 tau1) w + tau0 c^2)   -- no second exponential, no extra reciprocal.
    // 40 of the 96 FP64 instructions of a stage's gate rates go away (identical in exact arithmetic; the rates stay within a
    // few ulp of the tanh definition: tests/test_gpu_math.py).  u saturates at 2^+-250 (u^4 stays finite), where every
    // tanh is +-1 to far below half an ulp.
    static __device__ __forceinline__ void gates_shared_exp(double V, double m, double h, double n, double Fg[3]) {
        const double u = exp_affine_sat_k<250>(V, 1.0 / 15.0, 55.0 / 15.0);
        const double w = u * u;
        {   // m: (V_a, dV_a, tau0, tau1) = (-40, 15, 0.1, 0.4)
            const double e = 0x1.152aaa3bf81ccp-3 * w;                       // e^{-2} w
            const double q = e + 1.0;
            const double den = fma(e, fma(e, 0.1, 2.0 * 0.1 + 4.0 * 0.4), 0.1);
            Fg[0] = div_series(fma(-m, q, e) * q, den);
        }
        {   // h: (-60, -15, 1, 7)
            constexpr double c = 0x1.06de9bcee72dep-1;                       // e^{-2/3}
            const double Q = c + w;
            const double den = fma(w, fma(w, 1.0, c * (2.0 * 1.0 + 4.0 * 7.0)), 1.0 * c * c);
            Fg[1] = div_series(fma(-h, Q, c) * Q, den);
        }
        {   // n: (-55, 30, 1, 5)
            const double q = u + 1.0;
            const double den = fma(u, fma(u, 1.0, 2.0 * 1.0 + 4.0 * 5.0), 1.0);
            Fg[2] = div_series(fma(-n, q, u) * q, den);
        }
    }
    // fp32: the same sharing; u saturates at 2^+-30 (u^4 finite in fp32; tanh = +-1 to 2^-29, below half an fp32 ulp)
    static __device__ __forceinline__ void gates_shared_exp_f(float V, float m, float h, float n, float Fg[3]) {
        const float u = expf_sat_k<30>(fmaf(V, 1.0f / 15.0f, 55.0f / 15.0f));
        const float w = u * u;
        {
            const float e = 0.135335283236612692f * w;
            const float q = e + 1.0f;
            const float den = fmaf(e, fmaf(e, 0.1f, 2.0f * 0.1f + 4.0f * 0.4f), 0.1f);
            Fg[0] = divf_fast(fmaf(-m, q, e) * q, den);
        }
        {
            constexpr float c = 0.513417119032592027f;
            const float Q = c + w;
            const float den = fmaf(w, fmaf(w, 1.0f, c * 30.0f), c * c);
            Fg[1] = divf_fast(fmaf(-h, Q, c) * Q, den);
        }
        {
            const float q = u + 1.0f;
            const float den = fmaf(u, fmaf(u, 1.0f, 22.0f), 1.0f);
            Fg[2] = divf_fast(fmaf(-n, q, u) * q, den);
        }
    }
    static __device__ __forceinline__ void rhs(const R x[4], const R* __restrict__ p, R inv_C, R I, R F[4]) {
        F[0] = rhs_V(x, p, inv_C, I);
        rhs_gates(x, F + 1);
    }
    // The first RK4 stage evaluates the gate rates at x itself: they do not depend on the parameters, so a parameter
    // move (row A4: same x, seven different p per sweep) can reuse them.  NK values per site are cached by the tile engine.
    static constexpr int NK = 3;
    static __device__ __forceinline__ void stage1_cache(const R x[4], R kg[3]) { rhs_gates(x, kg); }
    // Quantities that depend only on (p, dt): computed once per parameter vector, not once per site.
    struct Prep { R inv_C, hdt, dt6; };
    static __device__ __forceinline__ Prep prepare(const R* __restrict__ p, R dt) {
        Prep q;
        if constexpr (sizeof(R) == 8) q.inv_C = div_fast(1.0, p[6]);
        else q.inv_C = 1.0f / p[6];
        q.hdt = R(0.5) * dt;
        q.dt6 = dt / R(6);
        return q;
    }
    // The same for a parameter move that changes entry l only: 1/C has to be recomputed for l = 6 (C) alone -- the division
    // is the first thing on the dependent chain of the evaluation.
    static __device__ __forceinline__ Prep prepare_move(const Prep& cur, const R* __restrict__ p_new, R dt, int l) {
        if (l == NP - 1) return prepare(p_new, dt);
        return cur;
    }
    static constexpr R kVmax = sizeof(R) == 8 ? R(1e8) : R(1e6);
    // Domain guard of the branch-free gates: a stage voltage beyond +-1e8 mV (fp32: 1e6 mV) or NaN makes the whole increment
    // NaN, i.e. the proposal is rejected; inside the guard the gates saturate exactly like tanh.
    // kg_in: stage-1 gate rates computed earlier at this same x (bit-identical to recomputing them); kg_out: receives them
    template <bool IN, bool OUT>
    static __device__ __forceinline__ void increment_k(const R x[4], const R* __restrict__ p, const Prep& q, R I0, R I1, R dt, R g[4],
                                                       const R* kg_in, R* kg_out) {
        const R Ih = R(0.5) * (I0 + I1);
        R k[4], xs[4], acc[4];
        bool sane = true;
        if constexpr (IN) {
            k[0] = rhs_V(x, p, q.inv_C, I0);
#pragma unroll
            for (int a = 0; a < 3; ++a) k[1 + a] = kg_in[a];
        } else rhs(x, p, q.inv_C, I0, k);
        if constexpr (OUT) {
#pragma unroll
            for (int a = 0; a < 3; ++a) kg_out[a] = k[1 + a];
        }
        sane = sane && fabs(x[0]) < kVmax;
#pragma unroll
        for (int a = 0; a < 4; ++a) { acc[a] = k[a]; xs[a] = x[a] + q.hdt * k[a]; }
        rhs(xs, p, q.inv_C, Ih, k);
        sane = sane && fabs(xs[0]) < kVmax;
#pragma unroll
        for (int a = 0; a < 4; ++a) { acc[a] += R(2) * k[a]; xs[a] = x[a] + q.hdt * k[a]; }
        rhs(xs, p, q.inv_C, Ih, k);
        sane = sane && fabs(xs[0]) < kVmax;
#pragma unroll
        for (int a = 0; a < 4; ++a) { acc[a] += R(2) * k[a]; xs[a] = x[a] + dt * k[a]; }
        rhs(xs, p, q.inv_C, I1, k);
        sane = sane && fabs(xs[0]) < kVmax;
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            g[a] = q.dt6 * (acc[a] + k[a]);
            g[a] = sane ? g[a] : (R)__longlong_as_double(0x7FF8000000000000ll);
        }
    }
    static __device__ __forceinline__ void increment(const R x[4], const R* __restrict__ p, const Prep& q, R I0, R I1, R dt, R g[4]) {
        increment_k<false, false>(x, p, q, I0, I1, dt, g, nullptr, nullptr);
    }
    static __device__ __forceinline__ void increment(const R x[4], const R* __restrict__ p, R I0, R I1, R dt, R g[4]) {
        increment(x, p, prepare(p, dt), I0, I1, dt, g);
    }
    // The parameters enter dV/dt LINEARLY through NTH monomials (Eq. 11; the gate equations hold none):
    //   (dt/2) F_V(x, p; I) = theta(p) . phi(x, I),  theta = (1, gNa, gNa ENa, gK, gK EK, gL, gL EL) / C,
    //                                                phi = (dt/2) (I, -m^3 h V, m^3 h, -n^4 V, n^4, -V, 1).
    // With the trapezoid rule (Eq. 7) every V residual is d_n - theta . (phi_n + phi_{n+1}), so the action is a
    // quadratic form in theta whose coefficients are sums over the path that do NOT depend on p: one reduction of those sums
    // per sweep decides all parameter moves (pimc_tile_kernel.cuh, "sufficient statistics").  Always in double.
    static constexpr int NTH = 7;
    // which monomials a move of parameter l changes (bit j = theta_j); a move of C (l = 6) changes 1/C and with it all of them
    static __host__ __device__ constexpr unsigned theta_mask(int l) {
        return l == 0 ? 0x06u : l == 1 ? 0x18u : l == 2 ? 0x60u : l == 3 ? 0x04u : l == 4 ? 0x10u : l == 5 ? 0x40u : 0x7Fu;
    }
    static __device__ __forceinline__ double theta_pre(const R* __restrict__ p) { return 1.0 / (double)p[6]; }
    static __device__ __forceinline__ void theta(const R* __restrict__ p, double th[7]) { theta_from(p, theta_pre(p), th); }
    static __device__ __forceinline__ void theta_from(const R* __restrict__ p, double ic, double th[7]) {
        th[0] = ic; th[1] = (double)p[0] * ic; th[2] = (double)p[0] * (double)p[3] * ic; th[3] = (double)p[1] * ic;
        th[4] = (double)p[1] * (double)p[4] * ic; th[5] = (double)p[2] * ic; th[6] = (double)p[2] * (double)p[5] * ic;
    }
    static __device__ __forceinline__ void regressors(const R x[4], R I, double hdt, double ph[7]) {
        const double V = x[0], m = x[1], h = x[2], n = x[3];
        const double m3h = m * m * m * h, n2 = n * n, n4 = n2 * n2;
        ph[0] = hdt * (double)I; ph[1] = -hdt * m3h * V; ph[2] = hdt * m3h; ph[3] = -hdt * n4 * V; ph[4] = hdt * n4; ph[5] = -hdt * V; ph[6] = hdt;
    }
    // Trapezoid discretisation (Eq. 7): the cached quantity is c = (dt/2) F(x, p; I)
    static __device__ __forceinline__ void half_rhs(const R x[4], const R* __restrict__ p, const Prep& q, R I, R c[4]) {
        R F[4];
        rhs(x, p, q.inv_C, I, F);
        bool sane = true;
        sane = fabs(x[0]) < kVmax;
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            c[a] = q.hdt * F[a];
            c[a] = sane ? c[a] : (R)__longlong_as_double(0x7FF8000000000000ll);
        }
    }
};

template <typename R> using HHModel = HHModelK<R, 0>;
template <typename R> using HHClassicModel = HHModelK<R, 1>;

// ---------------------------------------------------------------------------------------------------
template <typename R, int D_> struct LinearModel {
    static constexpr int D = D_;
    static constexpr int NP = D_ * D_;
    static constexpr bool kTileMc = false;
    struct Prep {};
    static __device__ __forceinline__ Prep prepare(const R* __restrict__, R) { return Prep{}; }
    static __device__ __forceinline__ Prep prepare_move(const Prep&, const R* __restrict__, R, int) { return Prep{}; }
    // Trapezoid form of the linear model: F(x) = (A x - x)/dt, so c = (dt/2) F = (A x - x)/2
    static __device__ __forceinline__ void half_rhs(const R x[D_], const R* __restrict__ p, const Prep&, R, R c[D_]) {
#pragma unroll
        for (int a = 0; a < D_; ++a) {
            R f = R(0);
#pragma unroll
            for (int b = 0; b < D_; ++b) f += p[a * D_ + b] * x[b];
            c[a] = R(0.5) * (f - x[a]);
        }
    }
    static constexpr int NK = 0;                   // nothing parameter-independent worth caching
    static constexpr int NTH = 0;                  // no sufficient-statistics form of the parameter moves (tile engine keeps the per-move evaluation)
    static __host__ __device__ constexpr unsigned theta_mask(int) { return 0u; }
    static __device__ __forceinline__ double theta_pre(const R*) { return 0.0; }
    static __device__ __forceinline__ void theta_from(const R*, double, double*) {}
    static __device__ __forceinline__ R rhs_V(const R*, const R*, R, R) { return R(0); }
    static __device__ __forceinline__ void theta(const R*, double*) {}
    static __device__ __forceinline__ void regressors(const R*, R, double, double*) {}
    static __device__ __forceinline__ void stage1_cache(const R*, R*) {}
    template <bool IN, bool OUT>
    static __device__ __forceinline__ void increment_k(const R x[D_], const R* __restrict__ p, const Prep&, R I0, R I1, R dt, R g[D_], const R*, R*) {
        increment(x, p, I0, I1, dt, g);
    }
    static __device__ __forceinline__ void increment(const R x[D_], const R* __restrict__ p, const Prep&, R I0, R I1, R dt, R g[D_]) {
        increment(x, p, I0, I1, dt, g);
    }
    static __device__ __forceinline__ void increment(const R x[D_], const R* __restrict__ p, R, R, R, R g[D_]) {
#pragma unroll
        for (int a = 0; a < D_; ++a) {
            R f = R(0);
#pragma unroll
            for (int b = 0; b < D_; ++b) f += p[a * D_ + b] * x[b];
            g[a] = f - x[a];
        }
    }
};

}  // namespace pimc

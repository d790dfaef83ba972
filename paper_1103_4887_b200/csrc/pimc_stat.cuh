// Sufficient statistics of the trapezoid parameter moves, shared by the tile-resident and the global-memory engine.
//
// With the paper's trapezoid rule (Eq. 7) the V residual of term n -> n+1 is d_n - theta(p) . psi_n, where theta are the
// Model::NTH = 7 parameter monomials of PAPER.md:256-260 Eq. 11 and psi_n = phi_n + phi_{n+1} their regressors (Model::theta,
// Model::regressors), so
//   Delta-A(p -> p') = (Rf_V / 2) [ (theta' - theta)^T Q (theta' + theta) - 2 (theta' - theta) . b ],   Q = sum psi psi^T,  b = sum d psi.
// Q (28 entries, j <= k) and b (7) do not depend on p: 35 sums over the path per SWEEP decide every parameter move of the sweep.
#pragma once
#include <type_traits>

namespace pimc {

constexpr int kStatN = 35;
constexpr int kStatSlots = 40;                                     // packets per mailbox record (35 used)
constexpr int kStatCols = 36;                                      // product columns (35 used)
// statistic v is psi[kStatJ[v]] * (kStatK[v] < 7 ? psi[kStatK[v]] : d): first Q row by row (j <= k), then b
__device__ const signed char kStatJ[kStatCols] = {0, 0, 0, 0, 0, 0, 0, 1, 1, 1, 1, 1, 1, 2, 2, 2, 2, 2, 3, 3, 3, 3, 4, 4, 4, 5, 5, 6, 0, 1, 2, 3, 4, 5, 6, 0};
__device__ const signed char kStatK[kStatCols] = {0, 1, 2, 3, 4, 5, 6, 1, 2, 3, 4, 5, 6, 2, 3, 4, 5, 6, 3, 4, 5, 6, 4, 5, 6, 5, 6, 6, 7, 7, 7, 7, 7, 7, 7, 7};
__host__ __device__ constexpr int stat_q(int j, int k) { return j * 7 - j * (j - 1) / 2 + (k - j); }     // entry (j, k), j <= k, of Q
__host__ __device__ constexpr int stat_qs(int j, int k) { return j <= k ? stat_q(j, k) : stat_q(k, j); }

template <int N, class F> __device__ __forceinline__ void static_for(F&& f) {
    if constexpr (N > 0) { static_for<N - 1>(f); f(std::integral_constant<int, N - 1>{}); }
}

// The decisions of one sweep, in parameter order, from the totals S[35].  With v = Q theta - b for the CURRENT parameters,
//   Delta-A = (Rf_V / 2) sum_j dtheta_j (2 v_j + (Q dtheta)_j),  and on accept  v += Q dtheta;
// a move of parameter l changes the monomials Model::theta_mask(l) only (compile time: the loop over l is unrolled and branch-free,
// so everything that does not hang on the previous decision is hoisted).  s_in[l]: 0 frozen, 1 proposal out of bounds (rejected
// unevaluated), 2 to be evaluated; s_pl[l] the proposed value; s_logu[l * logu_stride] the log-uniform of the accept test.
// prm is updated in place; bit l of n_prop / n_acc: move l was proposed / accepted; dA_out[l] (NaN if not evaluated).  Returns
// whether any move was accepted.  Every thread that calls it with the same inputs takes the same decisions.
template <class Model, typename R>
__device__ __forceinline__ bool stat_decide(const double* S, R* prm, double half_rf, const int* s_in, const double* s_pl, const double* s_logu,
                                            int logu_stride, unsigned& n_prop, unsigned& n_acc, double* dA_out) {
    constexpr int NP = Model::NP;
    double ic = Model::theta_pre(prm);
    double th[7], vv[7];
    Model::theta_from(prm, ic, th);
#pragma unroll
    for (int j = 0; j < 7; ++j) {
        double row = -S[28 + j];
#pragma unroll
        for (int k = 0; k < 7; ++k) row = fma(S[stat_qs(j, k)], th[k], row);
        vv[j] = row;
    }
    bool changed = false;
    n_prop = 0u; n_acc = 0u;
    static_for<NP>([&](auto LC) {
        constexpr int l = decltype(LC)::value;
        constexpr unsigned mask = Model::theta_mask(l);
        const int st = s_in[l];
        const double pl = s_pl[l], logu = s_logu[l * logu_stride];
        R pp[NP];
#pragma unroll
        for (int k = 0; k < NP; ++k) pp[k] = (k == l) ? (R)pl : prm[k];
        const double ic2 = mask == 0x7Fu ? Model::theta_pre(pp) : ic;
        double th2[7], dth[7], qd[7];
        Model::theta_from(pp, ic2, th2);
#pragma unroll
        for (int j = 0; j < 7; ++j) dth[j] = (mask >> j & 1u) ? th2[j] - th[j] : 0.0;
#pragma unroll
        for (int j = 0; j < 7; ++j) {
            double r = 0.0;
#pragma unroll
            for (int k = 0; k < 7; ++k) if (mask >> k & 1u) r = fma(S[stat_qs(j, k)], dth[k], r);
            qd[j] = r;
        }
        double acc = 0.0;
#pragma unroll
        for (int j = 0; j < 7; ++j) if (mask >> j & 1u) acc = fma(dth[j], fma(2.0, vv[j], qd[j]), acc);
        const double dA = half_rf * acc;
        const bool accept = st == 2 && logu < -dA;
#pragma unroll
        for (int j = 0; j < 7; ++j) {
            vv[j] = accept ? vv[j] + qd[j] : vv[j];
            if (mask >> j & 1u) th[j] = accept ? th2[j] : th[j];
        }
        ic = accept ? ic2 : ic;
        changed = changed || accept;
        prm[l] = accept ? (R)pl : prm[l];
        n_prop |= (st != 0 ? 1u : 0u) << l;
        n_acc |= (accept ? 1u : 0u) << l;
        dA_out[l] = st == 2 ? dA : __longlong_as_double(0x7FF8000000000000ll);
    });
    return changed;
}

}  // namespace pimc

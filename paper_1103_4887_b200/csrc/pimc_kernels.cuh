// Device side of libpimc: the persistent sweep kernel (rows A2-A6 of SURVEY.md §8(a)) and small helpers.
//
// Work decomposition.  A chain's M+1 time steps are cut into G contiguous tiles of `tile` sites (tile even,
// so every tile starts on an even site); tile b of chain c is CTA c*G + b.  Inside a half-sweep every
// site of one parity is independent, so the threads of a CTA stride over the tile's
// sites of that parity.  The whole pimc_sweep call is ONE launch: the CTA loops over sweeps; between
// half-sweeps it only has to agree with its two neighbour tiles (row A3), not with the whole grid:
//   * the even half-sweep of tile b reads x,g of site s-1  (last written by tile b-1's odd half-sweep),
//   * the odd  half-sweep of tile b reads x   of site e    (last written by tile b+1's even half-sweep),
// so each CTA publishes a monotonically increasing half-sweep count with a release store and the
// neighbour polls it with an acquire load.  Parameter moves need one scalar
// all-reduce per parameter: every CTA publishes its partial Delta-A, then every CTA sums all G partials in
// index order, so all CTAs take the same decision from bit-identical totals without a broadcast step
// (replaces the paper's second, single-thread kernel).  The two cache copies + selector of PAPER.md:244
// are kept: g[cur] is current, g[cur^1] receives the proposal's increments, accept flips cur.
// With G = 1 (batched chains, one CTA per chain) there is no inter-CTA traffic at all.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "pimc_model.cuh"
#include "pimc_rng.cuh"
#include "pimc_stat.cuh"

namespace pimc {

constexpr int kMaxD = 4;
constexpr int kMaxNp = 16;
constexpr int kMaxThreads = 512;
constexpr int kMaxHistSel = 64;

template <typename R> struct SweepArgs {
    // problem
    int M, L, n_chains, G, tile, kind;
    double ln_beta0;      // simulated annealing of the dynamics term (Eq. 10): beta_k = exp(ln_beta0 (1 - k/n_cool)),
    unsigned long long n_cool, t_anneal;   //   k = t - t_anneal < n_cool, else 1; n_cool = 0 switches it off
    // step-size auto-tuning (GLOBAL engine): per-(site, component) and per-parameter step sizes; ws == nullptr
    // means the uniform widths wx / wp are in use
    double* ws;           // (C, M+1, D) state step sizes
    unsigned int* nacc_s; // (C, M+1, D) accepted changes since the last adjustment
    double* wpd;          // (C, Np) parameter step sizes
    unsigned int* nacc_p; // (C, Np)
    int tune;             // adjust every tune_skip-th sweep counted from t_tune
    unsigned long long tune_skip, t_tune;
    double f_acc, alpha;
    int update_mode;      // 0 = joint D-vector proposal per site (Fig. 1), 1 = one component at a time, D decisions per site (GLOBAL engine)
    int disc;             // model-error discretisation: 0 = explicit RK4 map, 1 = trapezoid rule (Eq. 7)
    int nc;               // cache entries per chain: M (disc 0: g_n, n <= M-1) or M + 1 (disc 1: c_n = (dt/2) F(x_n), n <= M)
    R dt, Rm, Rf[kMaxD], wx[kMaxD];
    double wp[kMaxNp];
    // device state (per chain, chains concatenated)
    R* x;                 // (C, M+1, D)
    R* g[2];              // (C, nc, D) x 2: step caches (ping-pong)
    R* kg;                // (C, M, NK): parameter-independent first-stage gate rates of every site (Model::stage1_cache; RK4 map only),
                          //   kept current by the site updates and reused by the seven parameter moves of a sweep (GLOBAL engine)
    const R* y;           // (C, M+1, L)
    const R* I;           // (C, M+1) or nullptr
    R* p;                 // (C, Np)
    int* cur;             // (C) which cache is current
    const double* lo;     // (C, Np)
    const double* hi;
    // statistics
    int accum;
    unsigned long long n_skip, t_enable;
    unsigned long long skip0;    // (t0 - t_enable) mod n_skip: the tile engine counts from here instead of dividing every sweep
    double *cx, *S1x, *S2x;      // (C, M+1, D)
    double *cp, *S1p, *S2p;      // (C, Np)
    unsigned long long* counters;  // (C, 2, D+Np) accepted, proposed
    int n_sel, nbins;
    const int* hsite; const int* hcomp; const double* hlo; const double* hhi; const double* hwidth;
    unsigned long long* hist;    // (C, n_sel, nbins+2)
    // debug trace of the last sweep (all nullptr = off)
    R* tr_dA; unsigned char* tr_acc; R* tr_xprop; R* tr_dAp; unsigned char* tr_accp; R* tr_pprop;
    // run
    unsigned long long t0, seed;
    long long n_sweeps;
    int do_states, do_params;
    // inter-CTA hand-off (G > 1)
    unsigned long long* hs_flag;  // (C, G) completed half-sweeps
    double* ar_val;               // (C, 2, G) partial Delta-A
    unsigned long long* ar_flag;  // (C, 2, G)
    unsigned long long* ar_epoch; // (C) all-reduce events performed so far (device-side bookkeeping)
    unsigned long long hs_base;
    // tile-resident engine (pimc_tile_kernel.cuh): halo depth, tagged-packet mailboxes, fault flag
    int h;
    unsigned long long* hx_words;   // (kTileMaxCtas, 2 sides, 2 slots, kHaloWordsPerSide)
    unsigned long long* hx_epoch;   // (C) halo exchanges performed so far
    unsigned long long* ar_words;   // (2 slots, kTileMaxCtas, kArSlotWords) Delta-A partials, one 128-byte line per CTA
    int* fault;                     // set to 1 if a hand-off was never delivered
    // optional record of the parameters at every accumulated sweep (pimc_param_trace; Fig. 4)
    R* ptrace;                      // (C, ptrace_cap, Np) or nullptr
    long long ptrace_cap;
    unsigned long long ptrace_n0;   // records written before this launch (= samples accumulated so far)
    int ar_hold;                    // SM clock ticks between publishing a Delta-A partial and the first poll of the others' (pimc_set_exchange)
    unsigned long long* st_words;   // (2 slots, kTileMaxCtas, 2 {partials, totals}, kStatSlots) 16-byte tagged packets: sufficient statistics of the
                                    //   trapezoid parameter moves (tile engine)
    // many-chain tile-resident engine (pimc_tilemc_kernel.cuh): the chains [mc_chain0, mc_chain0 + mc_nchains) of this wave, the
    // first tag of this launch's private tag range, and the per-(chain, tile) mailboxes
    int mc_chain0, mc_nchains;
    unsigned int mc_tag0;
    unsigned long long* mc_hx_words;   // (kMcMaxSlots, 2 sides, 2 buffers, kHaloWordsPerSide)
    unsigned long long* mc_ar_words;   // (2 buffers, kMcMaxSlots, kArSlotWords)
};

// ---- annealing multiplier of the model-error weights at sweep t (same closed form as the oracle; beta = 1 when off) ----
template <typename R> __device__ __forceinline__ double anneal_beta(const SweepArgs<R>& a, unsigned long long t) {
    if (a.n_cool == 0ull || t < a.t_anneal) return 1.0;
    const unsigned long long k = t - a.t_anneal;
    if (k >= a.n_cool) return 1.0;
    return exp_fast(a.ln_beta0 * (1.0 - (double)k / (double)a.n_cool));
}

// ---- step-size adjustment between two launches of the tile-resident engine ------------------
// Delta_i <- Delta_i [1 + alpha (N_acc,i / N_skip - f_acc)] for every (chain, site, component) and every parameter, counters
// reset: the same correctly rounded operations, in the same order, as the in-kernel adjustment of sweep_kernel.
static __global__ void tune_adjust_kernel(double* __restrict__ ws, unsigned int* __restrict__ nacc_s, size_t n_site_widths,
                                          double* __restrict__ wpd, unsigned int* __restrict__ nacc_p, size_t n_param_widths,
                                          double n_skip, double f_acc, double alpha) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_site_widths + n_param_widths; i += stride) {
        double* w = i < n_site_widths ? ws + i : wpd + (i - n_site_widths);
        unsigned int* na = i < n_site_widths ? nacc_s + i : nacc_p + (i - n_site_widths);
        const double rate = __ddiv_rn((double)*na, n_skip);
        *w = __dmul_rn(*w, __dadd_rn(1.0, __dmul_rn(alpha, __dsub_rn(rate, f_acc))));
        *na = 0u;
    }
}

// ---- memory-model helpers ------------------------------------------------------------------------
__device__ __forceinline__ void st_release_gpu(unsigned long long* p, unsigned long long v) {
    asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_acquire_gpu(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
// Poll a monotonically increasing counter until it reaches `need`.  Gives up (and raises the fault flag, pimc_fault) after
// kWaitSpinLimit polls, or soon after another CTA has given up: a safety net against hangs -- in a co-resident (cooperative)
// launch a hand-off cannot be lost.
constexpr unsigned long long kWaitSpinLimit = 20ull * 1000 * 1000;
__device__ __forceinline__ void wait_counter_ge(const unsigned long long* p, unsigned long long need, int* fault) {
    unsigned long long spins = 0;
    while (ld_acquire_gpu(p) < need) {
        if (++spins > kWaitSpinLimit) { atomicExch(fault, 1); break; }
        if ((spins & 0xFFFFull) == 0 && *reinterpret_cast<volatile int*>(fault) != 0) break;
    }
}
// Path and cache values may have been written by a neighbour CTA: read them from L2, never from a stale L1 line.
// CG = false (one CTA per chain: nobody else writes this chain) uses ordinary L1-cached loads, which the prefetches of the
// sweep loops can serve.
template <typename R, int D, bool CG = true> __device__ __forceinline__ void load_vec(const R* base, size_t site, R out[D]) {
    const R* q = base + site * D;
    if constexpr (!CG) {
        if constexpr (D == 4 && sizeof(R) == 8) {
            const double2 a = reinterpret_cast<const double2*>(q)[0], b = reinterpret_cast<const double2*>(q)[1];
            out[0] = a.x; out[1] = a.y; out[2] = b.x; out[3] = b.y;
        } else if constexpr (D == 4 && sizeof(R) == 4) {
            const float4 a = reinterpret_cast<const float4*>(q)[0];
            out[0] = a.x; out[1] = a.y; out[2] = a.z; out[3] = a.w;
        } else {
#pragma unroll
            for (int a = 0; a < D; ++a) out[a] = q[a];
        }
    } else if constexpr (D == 4 && sizeof(R) == 8) {
        const double2 a = __ldcg(reinterpret_cast<const double2*>(q));
        const double2 b = __ldcg(reinterpret_cast<const double2*>(q) + 1);
        out[0] = a.x; out[1] = a.y; out[2] = b.x; out[3] = b.y;
    } else if constexpr (D == 4 && sizeof(R) == 4) {
        const float4 a = __ldcg(reinterpret_cast<const float4*>(q));
        out[0] = a.x; out[1] = a.y; out[2] = a.z; out[3] = a.w;
    } else if constexpr (D == 2 && sizeof(R) == 8) {
        const double2 a = __ldcg(reinterpret_cast<const double2*>(q));
        out[0] = a.x; out[1] = a.y;
    } else {
#pragma unroll
        for (int a = 0; a < D; ++a) out[a] = __ldcg(q + a);
    }
}
__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }
template <typename R, int D> __device__ __forceinline__ void store_vec(R* base, size_t site, const R v[D]) {
    R* q = base + site * D;
    if constexpr (D == 4 && sizeof(R) == 8) {
        reinterpret_cast<double2*>(q)[0] = make_double2(v[0], v[1]);
        reinterpret_cast<double2*>(q)[1] = make_double2(v[2], v[3]);
    } else if constexpr (D == 4 && sizeof(R) == 4) {
        reinterpret_cast<float4*>(q)[0] = make_float4(v[0], v[1], v[2], v[3]);
    } else if constexpr (D == 2 && sizeof(R) == 8) {
        reinterpret_cast<double2*>(q)[0] = make_double2(v[0], v[1]);
    } else {
#pragma unroll
        for (int a = 0; a < D; ++a) q[a] = v[a];
    }
}

// ---- deterministic block sum: fixed xor tree inside a warp, then warps added in index order --------
__device__ __forceinline__ double block_sum(double v, double* red /* >= 32 doubles of shared memory */) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, off);
    const int warp = threadIdx.x >> 5, nwarps = (blockDim.x + 31) >> 5;
    if ((threadIdx.x & 31) == 0) red[warp] = v;
    __syncthreads();
    double tot = 0.0;
    for (int w = 0; w < nwarps; ++w) tot += red[w];
    __syncthreads();
    return tot;
}

// ---- proposals (Fig. 1 (a)) ---------------------------------------------------------------
template <typename R, int D>
__device__ __forceinline__ void propose_state(const SweepArgs<R>& a, unsigned long long t, uint32_t chain, uint32_t n,
                                              const R xn[D], R xp[D]) {
    const Words4 w = draw(a.seed, t, chain, n, kStreamStateProposal, 0);
    R wd[D];                                         // step sizes of this site: tuned per (site, component), else the uniform ones
#pragma unroll
    for (int c = 0; c < D; ++c) wd[c] = a.ws ? (R)a.ws[((size_t)chain * (a.M + 1) + n) * D + c] : a.wx[c];
    if (a.kind == 1) {   // uniform: x' = x + w (2u - 1)
#pragma unroll
        for (int c = 0; c < D; ++c) {
            if constexpr (sizeof(R) == 8) xp[c] = __dadd_rn(xn[c], __dmul_rn(wd[c], 2.0 * unit_open(w.w[c]) - 1.0));   // no FMA: bit-reproducible
            else xp[c] = __fadd_rn(xn[c], __fmul_rn(wd[c], __fsub_rn(__fmul_rn(2.0f, unit_openf(w.w[c])), 1.0f)));
        }
    } else {             // Gaussian: Box-Muller pairs from words (0,1) and (2,3)
        R z[4];
        if constexpr (sizeof(R) == 8) {
            normal_pair(unit_open(w.w[0]), unit_open(w.w[1]), z[0], z[1]);
            if constexpr (D > 2) normal_pair(unit_open(w.w[2]), unit_open(w.w[3]), z[2], z[3]);
        } else {
            normal_pair(unit_openf(w.w[0]), unit_openf(w.w[1]), z[0], z[1]);
            if constexpr (D > 2) normal_pair(unit_openf(w.w[2]), unit_openf(w.w[3]), z[2], z[3]);
        }
#pragma unroll
        for (int c = 0; c < D; ++c) {
            if constexpr (sizeof(R) == 8) xp[c] = __dadd_rn(xn[c], __dmul_rn(wd[c], z[c]));
            else xp[c] = __fadd_rn(xn[c], __fmul_rn(wd[c], z[c]));
        }
    }
}

template <typename R> __device__ __forceinline__ R log_accept_uniform(const SweepArgs<R>& a, unsigned long long t, uint32_t chain, uint32_t n, uint32_t block = 0) {
    const Words4 w = draw(a.seed, t, chain, n, kStreamStateAccept, block);
    if constexpr (sizeof(R) == 8) return log_fast(unit_open52(w.w[0], w.w[1]));
    else return logf(unit_openf(w.w[0]));
}

// ---- one Metropolis site update: Fig. 1 (a)-(i) ----------------------------------------------------------
template <class Model, typename R, bool CG = true>
__device__ __forceinline__ unsigned update_site(const SweepArgs<R>& a, const R* __restrict__ prm, unsigned long long t,
                                            uint32_t chain, int n, R* __restrict__ x, R* __restrict__ g, const R* __restrict__ y,
                                            const R* __restrict__ I, bool trace, size_t chain_site0, const R* __restrict__ Rfs,
                                            const typename Model::Prep& prep, R* __restrict__ kg) {
    constexpr int D = Model::D;
    constexpr int NK = Model::NK;
    R kgn[NK > 0 ? NK : 1];
    const int M = a.M;
    R xn[D], xfull[D], xp[D], gp[D];
    load_vec<R, D, CG>(x, n, xn);
    propose_state<R, D>(a, t, chain, (uint32_t)n, xn, xfull);
    // joint move: one pass with the whole proposal.  Component-wise moves: D passes; pass ai changes component ai only (same
    // draw as the joint move), is judged with the accept uniform of block ai, and the next pass starts from what it leaves.
    const int ncomp = a.update_mode == 1 ? D : 1;
    unsigned accepted_mask = 0;                 // bit c: a move that changed component c was accepted
#pragma unroll 1
    for (int ai = 0; ai < ncomp; ++ai) {
#pragma unroll
    for (int c = 0; c < D; ++c) xp[c] = (a.update_mode == 1 && c != ai) ? xn[c] : xfull[c];
    R dL = R(0), dR = R(0);     // left part (term n-1 -> n and measurement n) and right part (term n -> n+1), summed separately
    if (a.disc == 1) {
        // trapezoid rule, Fig. 1 (b)-(f) as printed: c' = (dt/2) F(x'_n) enters BOTH neighbouring terms; every residual is
        // (x_{k+1} - x_k) - c_k - c_{k+1}
        R cn[D];
        load_vec<R, D, CG>(g, n, cn);
        const R I0 = I ? __ldg(I + n) : R(0);
        Model::half_rhs(xp, prm, prep, I0, gp);
        if (n >= 1) {
            R xm[D], cm[D];
            load_vec<R, D, CG>(x, n - 1, xm);
            load_vec<R, D, CG>(g, n - 1, cm);
#pragma unroll
            for (int c = 0; c < D; ++c) {
                const R r_new = ((xp[c] - xm[c]) - cm[c]) - gp[c];
                const R r_old = ((xn[c] - xm[c]) - cm[c]) - cn[c];
                dL += R(0.5) * Rfs[c] * (r_new * r_new - r_old * r_old);
            }
#pragma unroll
            for (int l = 0; l < D; ++l) {
                if (l < a.L) {
                    const R yn = __ldg(y + (size_t)n * a.L + l);
                    const R d_new = yn - xp[l], d_old = yn - xn[l];
                    dL += R(0.5) * a.Rm * (d_new * d_new - d_old * d_old);
                }
            }
        }
        if (n <= M - 1) {
            R xq[D], cq[D];
            load_vec<R, D, CG>(x, n + 1, xq);
            load_vec<R, D, CG>(g, n + 1, cq);
#pragma unroll
            for (int c = 0; c < D; ++c) {
                const R r_new = ((xq[c] - xp[c]) - gp[c]) - cq[c];
                const R r_old = ((xq[c] - xn[c]) - cn[c]) - cq[c];
                dR += R(0.5) * Rfs[c] * (r_new * r_new - r_old * r_old);
            }
        }
    } else {
    if (n >= 1) {
        R xm[D], gm[D];
        load_vec<R, D, CG>(x, n - 1, xm);
        load_vec<R, D, CG>(g, n - 1, gm);
#pragma unroll
        for (int c = 0; c < D; ++c) {   // model-error term n-1 -> n
            const R r_new = (xp[c] - xm[c]) - gm[c];
            const R r_old = (xn[c] - xm[c]) - gm[c];
            dL += R(0.5) * Rfs[c] * (r_new * r_new - r_old * r_old);
        }
#pragma unroll
        for (int l = 0; l < D; ++l) {    // measurement term n (the action sums n = 1..M); the first L components are observed
            if (l < a.L) {
                const R yn = __ldg(y + (size_t)n * a.L + l);
                const R d_new = yn - xp[l], d_old = yn - xn[l];
                dL += R(0.5) * a.Rm * (d_new * d_new - d_old * d_old);
            }
        }
    }
    if (n <= M - 1) {
        R xq[D], gn[D];
        load_vec<R, D, CG>(x, n + 1, xq);
        load_vec<R, D, CG>(g, n, gn);
        const R I0 = I ? __ldg(I + n) : R(0), I1 = I ? __ldg(I + n + 1) : R(0);
        Model::template increment_k<false, (NK > 0)>(xp, prm, prep, I0, I1, a.dt, gp, nullptr, kgn);
#pragma unroll
        for (int c = 0; c < D; ++c) {   // model-error term n -> n+1
            const R r_new = (xq[c] - xp[c]) - gp[c];
            const R r_old = (xq[c] - xn[c]) - gn[c];
            dR += R(0.5) * Rfs[c] * (r_new * r_new - r_old * r_old);
        }
    }
    }
    const R dA = dL + dR;
    const R logu = log_accept_uniform<R>(a, t, chain, (uint32_t)n, (uint32_t)ai);
    const bool accept = logu < -dA;      // NaN or +inf rejects; dA <= 0 always accepts
    if (accept) {
        store_vec<R, D>(x, n, xp);
        if (n < a.nc) store_vec<R, D>(g, n, gp);
        if constexpr (NK > 0) {
            if (a.disc == 0 && n < a.M) {
#pragma unroll
                for (int c = 0; c < NK; ++c) kg[(size_t)n * NK + c] = kgn[c];
            }
        }
#pragma unroll
        for (int c = 0; c < D; ++c) xn[c] = xp[c];
        accepted_mask |= a.update_mode == 1 ? (1u << ai) : ((1u << D) - 1u);
    }
    if (trace) {
        const size_t gs = chain_site0 + (size_t)n;
        if (a.update_mode == 1) {          // trace entries per (site, component)
            R xa = R(0);
#pragma unroll
            for (int c = 0; c < D; ++c) xa = (c == ai) ? xfull[c] : xa;
            if (a.tr_dA) a.tr_dA[gs * D + ai] = dA;
            if (a.tr_acc) a.tr_acc[gs * D + ai] = accept ? 1 : 0;
            if (a.tr_xprop) a.tr_xprop[gs * D + ai] = xa;
        } else {
            if (a.tr_dA) a.tr_dA[gs] = dA;
            if (a.tr_acc) a.tr_acc[gs] = accept ? 1 : 0;
            if (a.tr_xprop) store_vec<R, D>(a.tr_xprop, gs, xp);
        }
    }
    }
    return accepted_mask;
}

// ---- the persistent sweep kernel ---------------------------------------------------------------------------
// SOLO = one CTA per chain (G == 1, batched chains): no other CTA ever writes this chain's arrays, so the loops use L1-cached
// loads and prefetch the lines of their NEXT pass (same thread, T sites further on) before working on the current one -- the
// profile of config 4 (profiles/r02_cfg4.md) had `long_scoreboard` on top: 21 % of all samples sat on the first uses of the
// loads of a parameter-move pass.
template <class Model, typename R, bool SOLO = false>
__global__ void __launch_bounds__(kMaxThreads) sweep_kernel(const SweepArgs<R> a) {
    constexpr bool CG = !SOLO;
    constexpr int D = Model::D;
    constexpr int NP = Model::NP;
    __shared__ double red[32];
    __shared__ R ps[NP];          // current parameters
    __shared__ R ps_prop[NP];     // parameters with the proposed entry
    __shared__ unsigned int s_pacc[NP], s_pprop[NP];
    __shared__ double wps[NP];            // parameter step sizes in use (every CTA of a chain keeps the same copy)
    __shared__ unsigned int s_ntune[NP];  // accepted parameter moves since the last adjustment
    __shared__ double bcast[4];
    __shared__ int s_cur;

    const int G = a.G, M = a.M, T = blockDim.x, tid = threadIdx.x;
    const uint32_t chain = blockIdx.x / G;
    const int b = blockIdx.x % G;
    const int s = b * a.tile;
    const int e = min(s + a.tile, M + 1);
    const size_t site0 = (size_t)chain * (M + 1);

    R* x = a.x + site0 * D;
    R* const g_a = a.g[0] + (size_t)chain * a.nc * D;
    R* const g_b = a.g[1] + (size_t)chain * a.nc * D;
    const R* y = a.y + site0 * a.L;
    const R* I = a.I ? a.I + site0 : nullptr;
    R* const kgc = a.kg + (size_t)chain * M * (Model::NK > 0 ? Model::NK : 1);
    unsigned long long* hs_flag = a.hs_flag + (size_t)chain * G;

    if (tid < NP) {
        ps[tid] = a.p[(size_t)chain * NP + tid]; s_pacc[tid] = 0; s_pprop[tid] = 0;
        wps[tid] = a.ws ? a.wpd[(size_t)chain * NP + tid] : a.wp[tid];
        s_ntune[tid] = a.ws ? a.nacc_p[(size_t)chain * NP + tid] : 0u;
    }
    if (tid == 0) s_cur = a.cur[chain];
    __syncthreads();
    int cur = s_cur;
    unsigned int n_acc_comp[D];                       // accepted moves per component class (A6)
#pragma unroll
    for (int c = 0; c < D; ++c) n_acc_comp[c] = 0;
    unsigned long long ar_count = a.ar_epoch[chain];   // all-reduce events this chain has performed so far
    unsigned long long n_rec = 0;                      // sweeps accumulated by this launch so far

    for (long long i = 0; i < a.n_sweeps; ++i) {
        const unsigned long long t = a.t0 + (unsigned long long)i;
        const bool trace = (i == a.n_sweeps - 1) && (a.tr_dA || a.tr_acc || a.tr_xprop || a.tr_dAp || a.tr_accp || a.tr_pprop);
        R Rfs[D];                                  // model-error weights in effect this sweep (annealing multiplier applied)
        {
            const double beta = anneal_beta(a, t);
#pragma unroll
            for (int c = 0; c < D; ++c) Rfs[c] = (R)(beta * (double)a.Rf[c]);
        }

        // ---------------- A2/A3: even half-sweep, then odd half-sweep ----------------
        const typename Model::Prep prep = Model::prepare(ps, a.dt);      // 1/C, dt/2, dt/6: once per sweep, not once per site
        if (a.do_states) {
            for (int parity = 0; parity < 2; ++parity) {
                if (G > 1) {
                    if (tid == 0) {
                        const unsigned long long need = a.hs_base + 2ull * (unsigned long long)i + (unsigned long long)parity;
                        if (parity == 0 && b > 0) wait_counter_ge(hs_flag + b - 1, need, a.fault);
                        if (parity == 1 && b < G - 1) wait_counter_ge(hs_flag + b + 1, need, a.fault);
                    }
                    __syncthreads();
                }
                for (int n = s + parity + 2 * tid; n < e; n += 2 * T)
                {
                    if constexpr (SOLO) {        // next pass of this thread: sites n' - 1 .. n' + 1 and their cache entries
                        const int np = n + 2 * T;
                        if (np < e) {
                            const R* gq = cur ? g_b : g_a;
                            prefetch_l1(x + (size_t)(np - 1) * D); prefetch_l1(x + (size_t)np * D); prefetch_l1(x + (size_t)min(np + 1, M) * D);
                            prefetch_l1(gq + (size_t)(np - 1) * D); prefetch_l1(gq + (size_t)min(np, a.nc - 1) * D);
                        }
                    }
                    const unsigned mask = update_site<Model, R, CG>(a, ps, t, chain, n, x, cur ? g_b : g_a, y, I, trace, site0, Rfs, prep, kgc);
#pragma unroll
                    for (int c = 0; c < D; ++c) n_acc_comp[c] += (mask >> c) & 1u;
                    if (a.ws && a.tune) {        // N_acc,i of the tuning rule: this thread is the only writer of its site
#pragma unroll
                        for (int c = 0; c < D; ++c) a.nacc_s[(site0 + (size_t)n) * D + c] += (mask >> c) & 1u;
                    }
                }
                __syncthreads();
                if (G > 1 && tid == 0)
                    st_release_gpu(hs_flag + b, a.hs_base + 2ull * (unsigned long long)i + (unsigned long long)parity + 1ull);
            }
        }

        // ---------------- A4: parameter moves, in sequence ----------------
        bool stat_done = false;
        if constexpr (SOLO && Model::NTH > 0) {
            // Trapezoid rule, one CTA per chain: ALL parameter moves of the sweep from one pass over the chain (sufficient statistics,
            // pimc_stat.cuh / DESIGN.md 6.1b) instead of one pass, with a model evaluation of every site, per parameter.
            if (a.do_params && a.disc == 1) {
                stat_done = true;
                __shared__ double st_part[(kMaxThreads / 32) * kStatCols];
                __shared__ double st_tot[kStatSlots];
                __shared__ double st_pl[NP], st_logu[NP];
                __shared__ int st_in[NP];
                if (tid < NP) {          // this sweep's proposals, bounds verdicts and log-uniforms: they do not depend on one another's decisions
                    const bool live = wps[tid] > 0.0;
                    double pl = (double)ps[tid], lu = 0.0;
                    int verdict = 0;
                    if (live) {
                        const Words4 w = draw(a.seed, t, chain, (uint32_t)tid, kStreamParam, 0);
                        double step;
                        if (a.kind == 1) step = __dmul_rn(wps[tid], 2.0 * unit_open(w.w[0]) - 1.0);
                        else { double z0, z1; normal_pair(unit_open(w.w[0]), unit_open(w.w[1]), z0, z1); step = __dmul_rn(wps[tid], z0); }
                        if constexpr (sizeof(R) == 8) pl = __dadd_rn((double)ps[tid], step);
                        else pl = (double)__fadd_rn(ps[tid], (float)step);
                        lu = log_fast(unit_open52(w.w[2], w.w[3]));
                        const double lo = a.lo[(size_t)chain * NP + tid], hi = a.hi[(size_t)chain * NP + tid];
                        verdict = (pl >= lo && pl <= hi) ? 2 : 1;
                    }
                    st_pl[tid] = pl; st_logu[tid] = lu; st_in[tid] = verdict;
                }
                // the 35 sums over the terms n -> n+1 of this thread's sites, in the order of its loop
                double acc[kStatN];
#pragma unroll
                for (int v = 0; v < kStatN; ++v) acc[v] = 0.0;
                const double hdt = (double)prep.hdt;
                for (int n = tid; n < M; n += T) {
                    R xn[D], xq[D];
                    load_vec<R, D, CG>(x, n, xn);
                    load_vec<R, D, CG>(x, n + 1, xq);
                    double f0[7], f1[7], psi[8];
                    Model::regressors(xn, I ? __ldg(I + n) : R(0), hdt, f0);
                    Model::regressors(xq, I ? __ldg(I + n + 1) : R(0), hdt, f1);
#pragma unroll
                    for (int k = 0; k < 7; ++k) psi[k] = f0[k] + f1[k];
                    psi[7] = (double)xq[0] - (double)xn[0];
#pragma unroll
                    for (int j = 0; j < 7; ++j) {
#pragma unroll
                        for (int k = j; k < 7; ++k) acc[stat_q(j, k)] = fma(psi[j], psi[k], acc[stat_q(j, k)]);
                        acc[28 + j] = fma(psi[j], psi[7], acc[28 + j]);
                    }
                }
                // block sums in a fixed order: xor tree inside a warp, then the warps in index order
#pragma unroll
                for (int v = 0; v < kStatN; ++v) {
                    double q = acc[v];
#pragma unroll
                    for (int off = 16; off > 0; off >>= 1) q += __shfl_xor_sync(0xFFFFFFFFu, q, off);
                    if ((tid & 31) == 0) st_part[(tid >> 5) * kStatCols + v] = q;
                }
                __syncthreads();
                if (tid < kStatN) {
                    double q = 0.0;
                    for (int wq = 0; wq < (T >> 5); ++wq) q += st_part[wq * kStatCols + tid];
                    st_tot[tid] = q;
                }
                __syncthreads();
                double S[kStatN], dAs[NP];
#pragma unroll
                for (int v = 0; v < kStatN; ++v) S[v] = st_tot[v];
                R prm[NP];
#pragma unroll
                for (int k = 0; k < NP; ++k) prm[k] = ps[k];
                unsigned n_prop = 0, n_acc = 0;
                const bool changed = stat_decide<Model, R>(S, prm, 0.5 * (double)Rfs[0], st_in, st_pl, st_logu, 1, n_prop, n_acc, dAs);
                __syncthreads();                         // everybody has read ps
                if (tid == 0) {
#pragma unroll
                    for (int l = 0; l < NP; ++l) {
                        ps[l] = prm[l];
                        if (n_acc >> l & 1u) s_ntune[l] += 1u;
                        s_pprop[l] += n_prop >> l & 1u;
                        s_pacc[l] += n_acc >> l & 1u;
                        if (trace) {
                            const bool frozen = !(n_prop >> l & 1u);
                            if (a.tr_dAp) a.tr_dAp[(size_t)chain * NP + l] = frozen ? (R)__longlong_as_double(0x7FF8000000000000ll) : (R)dAs[l];
                            if (a.tr_accp) a.tr_accp[(size_t)chain * NP + l] = (n_acc >> l & 1u) ? 1 : 0;
                            if (a.tr_pprop) a.tr_pprop[(size_t)chain * NP + l] = frozen ? prm[l] : (R)st_pl[l];
                        }
                    }
                }
                if (changed) {                           // the V entry of the cache under the final parameters (the gate entries hold no parameter)
                    const typename Model::Prep pq = Model::prepare(prm, a.dt);
                    R* gcur = cur ? g_b : g_a;
                    for (int n = tid; n <= M; n += T) {
                        R xn[D];
                        load_vec<R, D, CG>(x, n, xn);
                        const R c0 = pq.hdt * Model::rhs_V(xn, prm, pq.inv_C, I ? __ldg(I + n) : R(0));
                        gcur[(size_t)n * D] = fabs(xn[0]) < Model::kVmax ? c0 : (R)__longlong_as_double(0x7FF8000000000000ll);
                    }
                }
                __syncthreads();
            }
        }
        if (a.do_params && !stat_done) {
            for (int l = 0; l < NP; ++l) {
                if (!(wps[l] > 0.0)) continue;
                // one thread draws the proposal and the accept uniform; everybody needs p', log u and the bounds verdict
                if (tid == 0) {
                    const Words4 w = draw(a.seed, t, chain, (uint32_t)l, kStreamParam, 0);
                    double step;
                    if (a.kind == 1) step = __dmul_rn(wps[l], 2.0 * unit_open(w.w[0]) - 1.0);
                    else { double z0, z1; normal_pair(unit_open(w.w[0]), unit_open(w.w[1]), z0, z1); step = __dmul_rn(wps[l], z0); }
                    double pl;
                    if constexpr (sizeof(R) == 8) pl = __dadd_rn((double)ps[l], step);
                    else pl = (double)__fadd_rn(ps[l], (float)step);
                    const double lo = a.lo[(size_t)chain * NP + l], hi = a.hi[(size_t)chain * NP + l];
                    bcast[0] = pl;
                    bcast[1] = log_fast(unit_open52(w.w[2], w.w[3]));
                    bcast[2] = (pl >= lo && pl <= hi) ? 1.0 : 0.0;
                }
                if (tid < NP) ps_prop[tid] = ps[tid];
                __syncthreads();
                const double pl = bcast[0], logu = bcast[1];
                const bool inside = bcast[2] != 0.0;
                bool accept = false;
                double dA = __longlong_as_double(0x7FF8000000000000ll);   // NaN = not evaluated
                if (inside) {   // a proposal outside the bounds is rejected (without evaluating the model)
                    if (tid == 0) ps_prop[l] = (R)pl;
                    __syncthreads();
                    R* gcur = cur ? g_b : g_a;
                    R* galt = cur ? g_a : g_b;
                    double part = 0.0;
                    const int e_fwd = min(e, M);
                    if (a.disc == 1) {
                        // trapezoid rule: term n -> n+1 needs c'_n and c'_{n+1}; the thread of site n evaluates both (the field is
                        // one right-hand side, a quarter of an RK4 step) and stores c'_n (and c'_M with the last term)
                        const typename Model::Prep pq = Model::prepare(ps_prop, a.dt);
                        for (int n = s + tid; n < e_fwd; n += T) {
                            R xn[D], xq[D], cn[D], cq[D], cpn[D], cpq[D];
                            load_vec<R, D, CG>(x, n, xn);
                            load_vec<R, D, CG>(x, n + 1, xq);
                            load_vec<R, D, CG>(gcur, n, cn);
                            load_vec<R, D, CG>(gcur, n + 1, cq);
                            Model::half_rhs(xn, ps_prop, pq, I ? __ldg(I + n) : R(0), cpn);
                            Model::half_rhs(xq, ps_prop, pq, I ? __ldg(I + n + 1) : R(0), cpq);
                            store_vec<R, D>(galt, n, cpn);
                            if (n + 1 == M) store_vec<R, D>(galt, n + 1, cpq);
                            R acc = R(0);
#pragma unroll
                            for (int c = 0; c < D; ++c) {
                                const R d = xq[c] - xn[c];
                                const R r_new = (d - cpn[c]) - cpq[c], r_old = (d - cn[c]) - cq[c];
                                acc += R(0.5) * Rfs[c] * (r_new * r_new - r_old * r_old);
                            }
                            part += (double)acc;
                        }
                    } else {
                    const typename Model::Prep pq = Model::prepare(ps_prop, a.dt);
                    for (int n = s + tid; n < e_fwd; n += T) {
                        if constexpr (SOLO) {    // x_{n'+1} is the next lane's x_{n'}: one prefetch per array covers the warp's lines
                            const int np = n + T;
                            if (np < e_fwd) { prefetch_l1(x + (size_t)np * D); prefetch_l1(gcur + (size_t)np * D); prefetch_l1(kgc + (size_t)np * Model::NK); if (I) prefetch_l1(I + np); }
                        }
                        R xn[D], xq[D], gn[D], gp[D];
                        load_vec<R, D, CG>(x, n, xn);
                        load_vec<R, D, CG>(x, n + 1, xq);
                        load_vec<R, D, CG>(gcur, n, gn);
                        const R I0 = I ? __ldg(I + n) : R(0), I1 = I ? __ldg(I + n + 1) : R(0);
                        constexpr int NK = Model::NK;
                        R kk[NK > 0 ? NK : 1];
                        if constexpr (NK > 0) {
#pragma unroll
                            for (int c = 0; c < NK; ++c) kk[c] = CG ? __ldcg(kgc + (size_t)n * NK + c) : kgc[(size_t)n * NK + c];
                        }
                        Model::template increment_k<(NK > 0), false>(xn, ps_prop, pq, I0, I1, a.dt, gp, kk, nullptr);
                        store_vec<R, D>(galt, n, gp);
                        R acc = R(0);
#pragma unroll
                        for (int c = 0; c < D; ++c) {
                            const R d = xq[c] - xn[c];
                            const R r_new = d - gp[c], r_old = d - gn[c];
                            acc += R(0.5) * Rfs[c] * (r_new * r_new - r_old * r_old);
                        }
                        part += (double)acc;
                    }
                    }
                    dA = block_sum(part, red);
                    if (G > 1) {   // all-gather of the G partials, summed in index order by every CTA
                        const int slot = (int)(ar_count & 1ull);
                        double* val = a.ar_val + ((size_t)chain * 2 + slot) * G;
                        unsigned long long* flg = a.ar_flag + ((size_t)chain * 2 + slot) * G;
                        if (tid == 0) {
                            val[b] = dA;
                            st_release_gpu(flg + b, ar_count + 1ull);
                        }
                        double mine = 0.0;
                        for (int j = tid; j < G; j += T) {
                            wait_counter_ge(flg + j, ar_count + 1ull, a.fault);
                            mine += __ldcg(val + j);
                        }
                        dA = block_sum(mine, red);
                        ar_count += 1ull;
                    }
                    accept = logu < -dA;
                    if (accept) cur ^= 1;
                }
                if (tid == 0) {
                    if (accept) { ps[l] = (R)pl; s_ntune[l] += 1u; }
                    if (b == 0) {
                        s_pprop[l] += 1;
                        if (accept) s_pacc[l] += 1;
                        if (trace) {
                            if (a.tr_dAp) a.tr_dAp[(size_t)chain * NP + l] = (R)dA;
                            if (a.tr_accp) a.tr_accp[(size_t)chain * NP + l] = accept ? 1 : 0;
                            if (a.tr_pprop) a.tr_pprop[(size_t)chain * NP + l] = (R)pl;
                        }
                    }
                }
                __syncthreads();
            }
            if (trace && b == 0 && tid == 0) {
                for (int l = 0; l < NP; ++l)
                    if (!(wps[l] > 0.0)) {
                        if (a.tr_dAp) a.tr_dAp[(size_t)chain * NP + l] = (R)__longlong_as_double(0x7FF8000000000000ll);
                        if (a.tr_accp) a.tr_accp[(size_t)chain * NP + l] = 0;
                        if (a.tr_pprop) a.tr_pprop[(size_t)chain * NP + l] = ps[l];
                    }
            }
        }

        // ---------------- A5: running moments and histograms ----------------
        if (a.accum && ((t - a.t_enable) % a.n_skip) == 0ull) {
            // own sites only; they were last written by this CTA (visible after the barriers above)
            // four elements per thread per pass with all loads issued before the first store (the arrays do not alias): the
            // loop is bound by the L2/HBM round trip of its read-modify-writes, not by arithmetic
            {
                const R* __restrict__ xr = x;
                const double* __restrict__ cxr = a.cx + site0 * D;
                double* __restrict__ S1r = a.S1x + site0 * D;
                double* __restrict__ S2r = a.S2x + site0 * D;
                const int lo_i = s * D, hi_i = e * D;
                int i0 = lo_i + tid;
                for (; i0 + 3 * T < hi_i; i0 += 4 * T) {
                    const double x0 = (double)__ldcg(xr + i0), x1 = (double)__ldcg(xr + i0 + T), x2 = (double)__ldcg(xr + i0 + 2 * T), x3 = (double)__ldcg(xr + i0 + 3 * T);
                    const double c0 = cxr[i0], c1 = cxr[i0 + T], c2 = cxr[i0 + 2 * T], c3 = cxr[i0 + 3 * T];
                    const double p0 = S1r[i0], p1 = S1r[i0 + T], p2 = S1r[i0 + 2 * T], p3 = S1r[i0 + 3 * T];
                    const double q0 = S2r[i0], q1 = S2r[i0 + T], q2 = S2r[i0 + 2 * T], q3 = S2r[i0 + 3 * T];
                    const double d0 = x0 - c0, d1 = x1 - c1, d2 = x2 - c2, d3 = x3 - c3;
                    S1r[i0] = p0 + d0; S1r[i0 + T] = p1 + d1; S1r[i0 + 2 * T] = p2 + d2; S1r[i0 + 3 * T] = p3 + d3;
                    S2r[i0] = q0 + d0 * d0; S2r[i0 + T] = q1 + d1 * d1; S2r[i0 + 2 * T] = q2 + d2 * d2; S2r[i0 + 3 * T] = q3 + d3 * d3;
                }
                for (; i0 < hi_i; i0 += T) {
                    const double d = (double)__ldcg(xr + i0) - cxr[i0];
                    S1r[i0] += d;
                    S2r[i0] += d * d;
                }
            }
            if (b == 0 && tid < NP) {
                const size_t gi = (size_t)chain * NP + tid;
                const double d = (double)ps[tid] - a.cp[gi];
                a.S1p[gi] += d;
                a.S2p[gi] += d * d;
                const unsigned long long rec = a.ptrace_n0 + n_rec;
                if (a.ptrace && rec < (unsigned long long)a.ptrace_cap) a.ptrace[((size_t)chain * a.ptrace_cap + rec) * NP + tid] = ps[tid];
            }
            n_rec += 1ull;
            for (int sel = tid; sel < a.n_sel; sel += T) {
                const int site = a.hsite[sel], comp = a.hcomp[sel];
                const bool mine = site < 0 ? (b == 0) : (site >= s && site < e);
                if (mine) {
                    const double v = site < 0 ? (double)ps[comp] : (double)__ldcg(x + (size_t)site * D + comp);
                    unsigned long long* bins = a.hist + ((size_t)chain * a.n_sel + sel) * (size_t)(a.nbins + 2);
                    const double lo = a.hlo[sel], hi = a.hhi[sel];
                    int bin;
                    if (!(v >= lo)) bin = 0;
                    else if (v >= hi) bin = a.nbins + 1;
                    else {
                        long long q = (long long)floor((v - lo) / a.hwidth[sel]);
                        if (q >= a.nbins) q = a.nbins - 1;
                        bin = 1 + (int)q;
                    }
                    bins[bin] += 1ull;     // one owner thread per selection: no atomics needed
                }
            }
            __syncthreads();   // the next half-sweep overwrites x
        }

        // ---------------- step-size adjustment, every tune_skip-th sweep while tuning ----------------
        // Delta_i <- Delta_i [1 + alpha (N_acc,i / N_skip - f_acc)]; written without FMA contraction, so that the step sizes
        // (and with them the proposals) stay bit-identical to the oracle's
        if (a.ws && a.tune && ((t - a.t_tune + 1ull) % a.tune_skip) == 0ull) {
            __syncthreads();
            const double ns = (double)a.tune_skip;
            for (int idx = s * D + tid; idx < e * D; idx += T) {
                const size_t gi = site0 * D + (size_t)idx;
                const double rate = __ddiv_rn((double)a.nacc_s[gi], ns);
                a.ws[gi] = __dmul_rn(a.ws[gi], __dadd_rn(1.0, __dmul_rn(a.alpha, __dsub_rn(rate, a.f_acc))));
                a.nacc_s[gi] = 0u;
            }
            if (tid < NP) {
                const double rate = __ddiv_rn((double)s_ntune[tid], ns);
                wps[tid] = __dmul_rn(wps[tid], __dadd_rn(1.0, __dmul_rn(a.alpha, __dsub_rn(rate, a.f_acc))));
                s_ntune[tid] = 0u;
            }
            __syncthreads();
        }
    }

    // ---------------- A6 + state write-back ----------------
    {
        double acc_total[D];
#pragma unroll
        for (int c = 0; c < D; ++c) acc_total[c] = block_sum((double)n_acc_comp[c], red);   // exact: counts < 2^53
        if (tid == 0) {
            unsigned long long* cnt = a.counters + (size_t)chain * 2 * (D + NP);
            unsigned long long prop_u = 0;
            if (a.do_states) prop_u = (unsigned long long)(e - s) * (unsigned long long)a.n_sweeps;
#pragma unroll
            for (int c = 0; c < D; ++c) {
                const unsigned long long acc_u = (unsigned long long)acc_total[c];
                if (acc_u) atomicAdd(cnt + c, acc_u);
                if (prop_u) atomicAdd(cnt + (D + NP) + c, prop_u);
            }
            if (b == 0) {
                for (int l = 0; l < NP; ++l) {
                    cnt[D + l] += s_pacc[l];
                    cnt[(D + NP) + D + l] += s_pprop[l];
                    a.p[(size_t)chain * NP + l] = ps[l];
                    if (a.ws) { a.wpd[(size_t)chain * NP + l] = wps[l]; a.nacc_p[(size_t)chain * NP + l] = s_ntune[l]; }
                }
                a.cur[chain] = cur;
                a.ar_epoch[chain] = ar_count;
            }
        }
    }
}

// ---- A0: (re)build the step cache of every chain ---------------------------------------------------------
template <class Model, typename R>
__global__ void build_cache_kernel(const R* __restrict__ x, const R* __restrict__ I, const R* __restrict__ p, R* __restrict__ g,
                                   int M, int n_chains, R dt, int disc, R* __restrict__ kg) {
    constexpr int D = Model::D;
    constexpr int NP = Model::NP;
    const int nc = disc == 1 ? M + 1 : M;          // entries per chain
    const size_t total = (size_t)n_chains * nc;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        const size_t chain = idx / nc;
        const int n = (int)(idx % nc);
        const R* prm = p + chain * NP;
        R xn[D], gn[D];
#pragma unroll
        for (int c = 0; c < D; ++c) xn[c] = x[(chain * (M + 1) + n) * D + c];
        const R I0 = I ? I[chain * (M + 1) + n] : R(0), I1 = (I && n < M) ? I[chain * (M + 1) + n + 1] : R(0);
        if (disc == 1) Model::half_rhs(xn, prm, Model::prepare(prm, dt), I0, gn);
        else {
            constexpr int NK = Model::NK;
            R kk[NK > 0 ? NK : 1];
            Model::template increment_k<false, (NK > 0)>(xn, prm, Model::prepare(prm, dt), I0, I1, dt, gn, nullptr, kk);
            if constexpr (NK > 0) {
#pragma unroll
                for (int c = 0; c < NK; ++c) kg[(chain * M + n) * NK + c] = kk[c];
            }
        }
#pragma unroll
        for (int c = 0; c < D; ++c) g[(chain * nc + n) * D + c] = gn[c];
    }
}

// ---- first-stage gate rates of every site from the current path (after launches of the tile-resident engine, which keeps its own copy
// in shared memory and does not write this array back) ----
template <class Model, typename R>
__global__ void build_stage1_kernel(const R* __restrict__ x, int M, int n_chains, R* __restrict__ kg) {
    constexpr int D = Model::D;
    constexpr int NK = Model::NK;
    if constexpr (NK > 0) {
        const size_t total = (size_t)n_chains * M;
        for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
            const size_t chain = idx / M;
            const int n = (int)(idx % M);
            R xn[D], kk[NK];
#pragma unroll
            for (int c = 0; c < D; ++c) xn[c] = x[(chain * (M + 1) + n) * D + c];
            Model::stage1_cache(xn, kk);
#pragma unroll
            for (int c = 0; c < NK; ++c) kg[idx * NK + c] = kk[c];
        }
    }
}

// ---- stand-alone step increment on arbitrary states (self-test entry) -------------------------------------
template <class Model, typename R>
__global__ void step_selftest_kernel(const R* __restrict__ x, const R* __restrict__ p, const R* __restrict__ I0,
                                     const R* __restrict__ I1, R dt, unsigned long long n, R* __restrict__ g) {
    constexpr int D = Model::D;
    constexpr int NP = Model::NP;
    const R* prm = p;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (unsigned long long)gridDim.x * blockDim.x) {
        R xn[D], gn[D];
#pragma unroll
        for (int c = 0; c < D; ++c) xn[c] = x[i * D + c];
        Model::increment(xn, prm, I0 ? I0[i] : R(0), I1 ? I1[i] : R(0), dt, gn);
#pragma unroll
        for (int c = 0; c < D; ++c) g[i * D + c] = gn[c];
    }
}

// ---- RNG self-test ------------------------------------------------------------------------------------------
static __global__ void rng_selftest_kernel(const uint32_t* __restrict__ ctrs, unsigned long long n, uint32_t k0, uint32_t k1,
                                    uint32_t* __restrict__ out, double* __restrict__ u_prop, double* __restrict__ u_acc,
                                    double* __restrict__ z) {
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (unsigned long long)gridDim.x * blockDim.x) {
        const Words4 w = philox4x32_10(ctrs[4 * i], ctrs[4 * i + 1], ctrs[4 * i + 2], ctrs[4 * i + 3], k0, k1);
        if (out) for (int j = 0; j < 4; ++j) out[4 * i + j] = w.w[j];
        if (u_prop) for (int j = 0; j < 4; ++j) u_prop[4 * i + j] = unit_open(w.w[j]);
        if (u_acc) u_acc[i] = unit_open52(w.w[0], w.w[1]);
        if (z) {
            normal_pair(unit_open(w.w[0]), unit_open(w.w[1]), z[4 * i], z[4 * i + 1]);
            normal_pair(unit_open(w.w[2]), unit_open(w.w[3]), z[4 * i + 2], z[4 * i + 3]);
        }
    }
}

// ---- elementary-function self-test: out (n,9) = exp, log, sqrt, sin, cos, 1/x, HH gate rates of m, h, n at (V = x, a = 0.3) ----
static __global__ void math_selftest_kernel(const double* __restrict__ x, unsigned long long n, double* __restrict__ out) {
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (unsigned long long)gridDim.x * blockDim.x) {
        const double v = x[i];
        const double av = fabs(v);
        double s, c;
        sincos_fast(fmin(av, 7.9), s, c);
        out[9 * i + 0] = exp_fast(fmin(fmax(v, -700.0), 700.0));
        out[9 * i + 1] = log_fast(fmax(av, 1e-300));
        out[9 * i + 2] = sqrt_fast(fmax(av, 1e-300));
        out[9 * i + 3] = s;
        out[9 * i + 4] = c;
        out[9 * i + 5] = rcp_fast(fmax(av, 1e-300));
        const double xg[4] = {v, 0.3, 0.3, 0.3};
        HHModel<double>::rhs_gates(xg, out + 9 * i + 6);          // the production gate code (one shared exponential)
    }
}

// ---- FP64 pipe probe: 8 independent FMA chains per thread, no memory traffic ------------------------------
static __global__ void fp64_peak_kernel(double* sink, int iters, double a, double b) {
    double v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = threadIdx.x * 1e-3 + i;
    for (int k = 0; k < iters; ++k) {
#pragma unroll
        for (int i = 0; i < 8; ++i) v[i] = fma(v[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += v[i];
    if (s == 1234.5) sink[0] = s;   // never true; keeps the chains alive
}

// ---- moments read-out: mean = c + S1/N, var = S2/N - (S1/N)^2 ---------------------------------------------
static __global__ void moments_kernel(const double* __restrict__ cx, const double* __restrict__ S1x, const double* __restrict__ S2x,
                               const double* __restrict__ cp, const double* __restrict__ S1p, const double* __restrict__ S2p,
                               size_t nx /* (M+1)*D */, int np, int n_chains, double N, double* __restrict__ out) {
    const size_t per_chain = 2 * nx + 2 * (size_t)np;
    const size_t total = (size_t)n_chains * (nx + np);
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        const size_t chain = idx / (nx + np), r = idx % (nx + np);
        double c, s1, s2;
        size_t o_mean, o_var;
        if (r < nx) {
            c = cx[chain * nx + r]; s1 = S1x[chain * nx + r]; s2 = S2x[chain * nx + r];
            o_mean = chain * per_chain + r; o_var = o_mean + nx;
        } else {
            const size_t l = r - nx;
            c = cp[chain * np + l]; s1 = S1p[chain * np + l]; s2 = S2p[chain * np + l];
            o_mean = chain * per_chain + 2 * nx + l; o_var = o_mean + np;
        }
        const double m1 = N > 0.0 ? s1 / N : 0.0;
        out[o_mean] = c + m1;
        out[o_var] = N > 0.0 ? s2 / N - m1 * m1 : 0.0;
    }
}

// ---- model errors eps_n and observation errors delta_n of the current path ------------------------------------
// eps_{n,a} = (x_{n+1,a} - x_{n,a}) - g_{n,a} (trapezoid: ... - c_n - c_{n+1}), n < M; delta_{n,l} = y_{n,l} - x_{n,l}, n >= 1, delta_0 = 0:
// the terms of the action as the sweep kernels form them.  Writes them out (eps_out / delta_out, either may be null) and/or adds
// them and their squares to the running sums acc = per chain [E1 (M,D), E2 (M,D), D1 (M+1,L), D2 (M+1,L)] (no FMA contraction:
// the sums are the oracle's bit for bit when the residuals are).
template <typename R>
__global__ void residual_kernel(const R* __restrict__ x, const R* __restrict__ g0, const R* __restrict__ g1, const int* __restrict__ cur,
                                const R* __restrict__ y, int M, int D, int L, int nc, int disc, int n_chains,
                                R* __restrict__ eps_out, R* __restrict__ delta_out, double* __restrict__ acc) {
    const size_t per_chain = (size_t)(M + 1);
    const size_t ne = (size_t)M * D, nd = (size_t)(M + 1) * L;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < (size_t)n_chains * per_chain; idx += (size_t)gridDim.x * blockDim.x) {
        const size_t chain = idx / per_chain;
        const int n = (int)(idx % per_chain);
        const R* xc = x + chain * per_chain * D;
        const R* gc = (cur[chain] ? g1 : g0) + chain * (size_t)nc * D;
        double* a_c = acc ? acc + chain * (2 * ne + 2 * nd) : nullptr;
        if (n < M) {
            for (int a = 0; a < D; ++a) {
                R r = (xc[(size_t)(n + 1) * D + a] - xc[(size_t)n * D + a]) - gc[(size_t)n * D + a];
                if (disc == 1) r -= gc[(size_t)(n + 1) * D + a];
                if (eps_out) eps_out[chain * ne + (size_t)n * D + a] = r;
                if (a_c) {
                    const double rd = (double)r;
                    a_c[(size_t)n * D + a] = __dadd_rn(a_c[(size_t)n * D + a], rd);
                    a_c[ne + (size_t)n * D + a] = __dadd_rn(a_c[ne + (size_t)n * D + a], __dmul_rn(rd, rd));
                }
            }
        }
        for (int l = 0; l < L; ++l) {
            const R d = n >= 1 ? y[(chain * per_chain + n) * L + l] - xc[(size_t)n * D + l] : R(0);
            if (delta_out) delta_out[chain * nd + (size_t)n * L + l] = d;
            if (a_c) {
                const double dd = (double)d;
                a_c[2 * ne + (size_t)n * L + l] = __dadd_rn(a_c[2 * ne + (size_t)n * L + l], dd);
                a_c[2 * ne + nd + (size_t)n * L + l] = __dadd_rn(a_c[2 * ne + nd + (size_t)n * L + l], __dmul_rn(dd, dd));
            }
        }
    }
}
// read-out of the running residual sums: mean = S1/N, var = S2/N - mean^2, same layout as acc
static __global__ void residual_stats_kernel(const double* __restrict__ acc, size_t ne, size_t nd, int n_chains, double N, double* __restrict__ out) {
    const size_t per = 2 * ne + 2 * nd;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < (size_t)n_chains * (ne + nd); idx += (size_t)gridDim.x * blockDim.x) {
        const size_t chain = idx / (ne + nd), r = idx % (ne + nd);
        const size_t o1 = r < ne ? r : 2 * ne + (r - ne), o2 = r < ne ? ne + r : 2 * ne + nd + (r - ne);
        const double m = N > 0.0 ? acc[chain * per + o1] / N : 0.0;
        out[chain * per + o1] = m;
        out[chain * per + o2] = N > 0.0 ? acc[chain * per + o2] / N - m * m : 0.0;
    }
}

// type conversion copy (double <- R) for re-centring the moments
template <typename R> __global__ void widen_kernel(const R* __restrict__ in, double* __restrict__ out, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) out[i] = (double)in[i];
}

}  // namespace pimc

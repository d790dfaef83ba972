// Tile-resident sweep kernel for MANY chains (engine PIMC_ENGINE_TILE_MC): rows A1-A6 of SURVEY.md §8(a) with several
// (chain, tile) pairs resident in the shared memory of every SM at once.
//
// Why.  tile_sweep_kernel (pimc_tile_kernel.cuh) holds ONE tile per SM: a half-sweep is one site-update deep and a parameter
// move ends in a grid-wide exchange, so one chain leaves the FP64 pipe idle while it waits (43 % / 27 % of the
// pipe in the state sweeps / parameter moves), and a single chain has nothing to fill those bubbles with.  Batched chains
// (BASELINE.json config 4: 128 chains x M = 8192; "shared memory" tiles, north_star (a) "one CTA-group per
// chain") do: here every CTA hosts NGRP independent GROUPS of 128 threads, each with its own chain tile (<= 256 sites incl.
// halos) in shared memory, its own named barrier and its own mailboxes.  While one group's partial sums cross L2, the other
// groups of the SM evaluate their model steps: four warps per scheduler, each from a different chain.
//   * a group's thread j owns the local site pair (2j, 2j+1): one site per half-sweep in the state sweeps (row A2), both
//     sites in a parameter move (row A4);
//   * the random numbers are drawn in line (Philox is stateless; with four warps per scheduler the other groups hide that
//     latency, so no producer warps and no ring buffer: 80 bytes per site less shared memory);
//   * halos as in the tile engine: updated redundantly, refreshed every h half-sweeps through tagged 8-byte packets (row A3);
//   * a parameter move's partial sums are gathered per CHAIN (G tiles), every group sums them in index order (row A4);
//   * chains that do not fit at once run in WAVES: the launcher starts one launch per wave of chains_per_wave chains, each
//     running all n sweeps of the pimc_sweep call on its chains.  Tags of a launch come from a range no other launch uses.
// Scope: the RK4-map discretisation with joint updates and uniform step sizes (the production path of configs 2-4); the
// launcher sends everything else (trapezoid rule, component-wise updates, debug trace, annealing, step-size tuning) to the
// other engines.
#pragma once
#include "pimc_tile_kernel.cuh"

namespace pimc {

constexpr int kMcGroup = 128;        // threads per group: four warps, one per scheduler
constexpr int kMcTileMax = 256;      // tile sites incl. halos per group: one (even, odd) pair per thread
constexpr int kMcPitch = 130;        // plane pitch: 128 pairs + the right neighbour of the last odd site
constexpr int kMcMaxSlots = 640;     // (chain, tile) pairs in flight per launch (mailbox slots): 148 SMs x 4 groups = 592 on a B200

__device__ __forceinline__ void bar_group(int grp) { asm volatile("bar.sync %0, 128;" ::"r"(grp + 1) : "memory"); }

// Deterministic sum over the 128 threads of a group with ONE named barrier (alternating buffers as in block_sum_db).
__device__ __forceinline__ double group_sum(double v, double* red /* [2][4] */, unsigned& phase, int grp, int j) {
    v = warp_sum_mma(v);
    double* buf = red + (phase & 1u) * 4;
    phase ^= 1u;
    if ((j & 31) == 0) buf[j >> 5] = v;
    bar_group(grp);
    return (buf[0] + buf[1]) + (buf[2] + buf[3]);
}

template <typename R> struct McSmem {
    double *S1, *S2;            // [2*D*P] running moments of the tile (fp64 always)
    double* red;                // [2][4]
    double *s_pl, *s_logu;      // [2 sets][kMaxNp] this sweep's proposed parameter values and log-uniforms
    int* s_in;                  // [2 sets][kMaxNp] 0 = frozen, 1 = out of bounds, 2 = to be evaluated
    unsigned int *s_pacc, *s_pprop;   // [kMaxNp]
    R *xs, *g0, *g1;            // [2*D*P]
    R* kg;                      // [2*NK*P]
    R *Is, *ys;                 // [kMcTileMax + 2], [kMcTileMax]
};

template <typename R> __host__ __device__ inline size_t mc_group_bytes(int D, int NK) {
    const size_t P = kMcPitch;
    const size_t dbl = 2 * 2 * D * P + 8 + 2 * kMaxNp + 2 * kMaxNp + kMaxNp + kMaxNp / 2 + kMaxNp / 2;
    const size_t real = 3 * 2 * D * P + 2 * (size_t)NK * P + (kMcTileMax + 4) + kMcTileMax;
    return (dbl * 8 + real * sizeof(R) + 15) & ~(size_t)15;
}

template <typename R> __device__ __forceinline__ McSmem<R> mc_carve(unsigned char* base, int D, int NK) {
    const size_t P = kMcPitch;
    McSmem<R> m;
    double* d = reinterpret_cast<double*>(base);
    m.S1 = d; d += 2 * D * P;
    m.S2 = d; d += 2 * D * P;
    m.red = d; d += 8;
    m.s_pl = d; d += 2 * kMaxNp;
    m.s_logu = d; d += 2 * kMaxNp;
    m.s_in = reinterpret_cast<int*>(d); d += kMaxNp;
    m.s_pacc = reinterpret_cast<unsigned int*>(d); d += kMaxNp / 2;
    m.s_pprop = reinterpret_cast<unsigned int*>(d); d += kMaxNp / 2;
    R* r = reinterpret_cast<R*>(d);
    m.xs = r; r += 2 * D * P;
    m.g0 = r; r += 2 * D * P;
    m.g1 = r; r += 2 * D * P;
    m.kg = r; r += 2 * (size_t)NK * P;
    m.Is = r; r += kMcTileMax + 4;
    m.ys = r; r += kMcTileMax;
    return m;
}

// A parameter move evaluates the thread's two tile sites in ONE branch-free block (sites beyond the tile compute on whatever the
// shared memory holds and are masked out of the sum), so that the compiler can interleave the two dependent chains: config 4's
// parameter moves 0.262 -> 0.229 ms per sweep of the 128 chains against one site after the other (measured).
template <class Model, typename R, int NGRP>
__global__ void __launch_bounds__(NGRP * kMcGroup, 1) tilemc_sweep_kernel(const SweepArgs<R> a) {
    constexpr int D = Model::D;
    constexpr int NP = Model::NP;
    constexpr int NK = Model::NK;
    constexpr int NKA = NK > 0 ? NK : 1;
    constexpr int P = kMcPitch;
    constexpr int L = 1;                           // one observed component (the launcher checks)
    constexpr int TG = kMcGroup;
    extern __shared__ __align__(16) unsigned char mc_smem_raw[];
    const int grp = threadIdx.x / TG, j = threadIdx.x % TG;
    const int G = a.G, M = a.M, h = a.h;
    // slot -> (chain of this wave, tile): consecutive slots go to different CTAs first, so that a partly filled wave still uses every SM
    const int slot = grp * (int)gridDim.x + (int)blockIdx.x;
    if (slot >= a.mc_nchains * G) return;          // idle group: no CTA-wide barrier anywhere below
    const int cw = slot / G, b = slot % G;
    const uint32_t chain = (uint32_t)(a.mc_chain0 + cw);
    const McSmem<R> sm = mc_carve<R>(mc_smem_raw + (size_t)grp * mc_group_bytes<R>(D, NK), D, NK);

    const int s = b * a.tile, e = min(s + a.tile, M + 1);
    const int s_ext = max(0, s - h), e_ext = min(M + 1, e + h), n_ext = e_ext - s_ext;   // s_ext is even (tile and h are)
    const size_t site0 = (size_t)chain * (M + 1);
    const bool edge_lo = s_ext == 0, edge_hi = e_ext == M + 1;
    const int mbox = cw * G + b;                   // mailbox index of this tile; its chain neighbours are mbox - 1, mbox + 1

    R* const gx = a.x + site0 * D;
    R* const gg0 = a.g[0] + (size_t)chain * a.nc * D;
    R* const gg1 = a.g[1] + (size_t)chain * a.nc * D;
    int cur = a.cur[chain];

    // ---- load the extended tile (site-major in global memory -> parity planes in shared memory) ----
    for (int idx = j; idx < n_ext * D; idx += TG) sm.xs[so<D>(idx / D, idx % D, P)] = gx[(size_t)s_ext * D + idx];
    {
        const R* gsrc = cur ? gg1 : gg0;
        R* gdst = cur ? sm.g1 : sm.g0;
        const int ng = min(e_ext, M) - s_ext;      // cache entries exist for n <= M-1
        for (int idx = j; idx < ng * D; idx += TG) gdst[so<D>(idx / D, idx % D, P)] = gsrc[(size_t)s_ext * D + idx];
    }
    for (int i = j; i <= n_ext; i += TG) {
        const int n = s_ext + i;
        sm.Is[i] = (a.I && n <= M) ? a.I[site0 + n] : R(0);
    }
    for (int idx = j; idx < n_ext * L; idx += TG) sm.ys[idx] = a.y[(site0 + s_ext) * L + idx];
    if (a.accum) {
        for (int idx = j; idx < n_ext * D; idx += TG) {
            const size_t gi = (site0 + s_ext) * D + idx;
            const int o = so<D>(idx / D, idx % D, P);
            sm.S1[o] = a.S1x[gi]; sm.S2[o] = a.S2x[gi];
        }
    }
    if (j < NP) { sm.s_pacc[j] = 0u; sm.s_pprop[j] = 0u; }
    R prm[NP];                                     // every thread keeps the (identical) parameter vector in registers
#pragma unroll
    for (int k = 0; k < NP; ++k) prm[k] = a.p[(size_t)chain * NP + k];
    // running moments of the parameters: thread j < NP of the chain's first tile keeps those of parameter j in registers
    double pS1 = 0.0, pS2 = 0.0, pcc = 0.0;
    if (a.accum && b == 0 && j < NP) {
        const size_t gi = (size_t)chain * NP + j;
        pS1 = a.S1p[gi]; pS2 = a.S2p[gi]; pcc = a.cp[gi];
    }

    unsigned int ar_count = 0, hx_count = 0;       // exchanges of this launch; tags = a.mc_tag0 + count + 1
    unsigned long long n_rec = 0;
    unsigned long long skip_ctr = a.skip0;
    unsigned int n_acc_state = 0;
    unsigned red_phase = 0;
    bar_group(grp);

    // first-stage rates of this thread's two tile sites from their current state (launch start and after every halo refresh)
    auto refresh_stage1 = [&]() {
        if constexpr (NK > 0) {
#pragma unroll 1
            for (int q = 0; q < 2; ++q) {
                if (2 * j + q < n_ext) {
                    R xn[D], kk[NKA];
                    lds_site<R, D>(sm.xs, q, j, P, xn);
                    Model::stage1_cache(xn, kk);
#pragma unroll
                    for (int c = 0; c < NK; ++c) sm.kg[(q * NK + c) * P + j] = kk[c];
                }
            }
        }
    };
    refresh_stage1();
    bar_group(grp);

    int k_phase = 0;                               // half-sweeps since the halos were last exact
    typename Model::Prep prep = Model::prepare(prm, a.dt);
    for (long long i = 0; i < a.n_sweeps; ++i) {
        const unsigned long long t = a.t0 + (unsigned long long)i;
        const int set = (int)(i & 1);
        const bool acc_now = a.accum && skip_ctr == 0ull;
        skip_ctr = (skip_ctr + 1ull == a.n_skip) ? 0ull : skip_ctr + 1ull;

        // ---- this sweep's parameter proposals p'_l = p_l + step_l, bounds verdicts and log-uniforms: they do not depend on the
        // state sweep or on the other parameters' decisions, so thread l posts them now and the moves start from three reads ----
        if (a.do_params && j < NP) {
            const bool live = a.wp[j] > 0.0;
            R pcur = R(0);
#pragma unroll
            for (int k = 0; k < NP; ++k) pcur = (k == j) ? prm[k] : pcur;
            double pl = (double)pcur, lu = 0.0;
            int verdict = 0;
            if (live) {
                const Words4 w = draw(a.seed, t, chain, (uint32_t)j, kStreamParam, 0);
                double step;
                if (a.kind == 1) step = __dmul_rn(a.wp[j], 2.0 * unit_open(w.w[0]) - 1.0);
                else { double z0, z1; normal_pair(unit_open(w.w[0]), unit_open(w.w[1]), z0, z1); step = __dmul_rn(a.wp[j], z0); }
                if constexpr (sizeof(R) == 8) pl = __dadd_rn((double)pcur, step);
                else pl = (double)__fadd_rn(pcur, (float)step);
                lu = log_fast(unit_open52(w.w[2], w.w[3]));
                const double lo = a.lo[(size_t)chain * NP + j], hi = a.hi[(size_t)chain * NP + j];
                verdict = (pl >= lo && pl <= hi) ? 2 : 1;
            }
            sm.s_pl[set * kMaxNp + j] = pl;
            sm.s_logu[set * kMaxNp + j] = lu;
            sm.s_in[set * kMaxNp + j] = verdict;
        }

        // ---------------- A2: even half-sweep, then odd half-sweep ----------------
        if (a.do_states) {
#pragma unroll 1
            for (int q = 0; q < 2; ++q) {
                const int k = k_phase + q + 1;           // half-sweeps run on the current halos, this one included
                const int iloc = 2 * j + q, n = s_ext + iloc;
                const bool ok = n <= M && iloc < n_ext && (edge_lo || iloc >= k) && (edge_hi || iloc < n_ext - k);
                if (ok) {
                    R st[D], logu;
                    produce_site<R, D>(a, t, chain, (uint32_t)n, a.wx, 1, st, 1, &logu);      // A1: in line
                    R* gc = cur ? sm.g1 : sm.g0;
                    const bool has_l = n >= 1, has_r = n <= M - 1;
                    const int jl = max(j - 1 + q, 0), jr = j + q;     // pair index of the left / right neighbour (plane 1 - q)
                    const int own = q * D * P + j, oth = (1 - q) * D * P;
                    R xn[D], xp[D], gp[D], kgn[NKA];
                    double mcc[D];                                   // moment centres: loaded before the model step, used after it
                    if (acc_now) {
                        const double* ccp = a.cx + (site0 + (size_t)n) * D;
#pragma unroll
                        for (int c = 0; c < D; ++c) mcc[c] = __ldg(ccp + c);
                    }
#pragma unroll
                    for (int c = 0; c < D; ++c) {
                        xn[c] = sm.xs[own + c * P];
                        if constexpr (sizeof(R) == 8) xp[c] = __dadd_rn(xn[c], st[c]);
                        else xp[c] = __fadd_rn(xn[c], st[c]);
                    }
                    Model::template increment_k<false, (NK > 0)>(xp, prm, prep, sm.Is[iloc], sm.Is[iloc + 1], a.dt, gp, nullptr, kgn);
                    R dL = R(0), dR = R(0);
#pragma unroll
                    for (int c = 0; c < D; ++c) {
                        const R xm = sm.xs[oth + c * P + jl], gm = gc[oth + c * P + jl];
                        const R r_new = (xp[c] - xm) - gm;
                        const R r_old = (xn[c] - xm) - gm;
                        dL += R(0.5) * a.Rf[c] * (r_new * r_new - r_old * r_old);
                    }
                    {
                        const R yn = sm.ys[iloc];
                        const R d_new = yn - xp[0], d_old = yn - xn[0];
                        dL += R(0.5) * a.Rm * (d_new * d_new - d_old * d_old);
                    }
#pragma unroll
                    for (int c = 0; c < D; ++c) {
                        const R xq = sm.xs[oth + c * P + jr], gn = gc[own + c * P];
                        const R r_new = (xq - xp[c]) - gp[c];
                        const R r_old = (xq - xn[c]) - gn;
                        dR += R(0.5) * a.Rf[c] * (r_new * r_new - r_old * r_old);
                    }
                    const R dA = (has_l ? dL : R(0)) + (has_r ? dR : R(0));
                    const bool accept = logu < -dA;
                    if (accept) {
#pragma unroll
                        for (int c = 0; c < D; ++c) sm.xs[own + c * P] = xp[c];
                        if (has_r) {
#pragma unroll
                            for (int c = 0; c < D; ++c) gc[own + c * P] = gp[c];
                        }
#pragma unroll
                        for (int c = 0; c < NK; ++c) sm.kg[(q * NK + c) * P + j] = kgn[c];
                    }
                    if (acc_now) {       // A5 for this site: its value is final for sweep t (parameter moves do not touch x)
#pragma unroll
                        for (int c = 0; c < D; ++c) {
                            const double d = (double)(accept ? xp[c] : xn[c]) - mcc[c];
                            sm.S1[own + c * P] += d;
                            sm.S2[own + c * P] += d * d;
                        }
                    }
                    n_acc_state += (accept && n >= s && n < e) ? 1u : 0u;
                }
                bar_group(grp);
            }
            k_phase += 2;
        } else bar_group(grp);                       // the posted proposals are read by every thread below

        // ---------------- A4: parameter moves, in sequence; the thread's two tile sites per move ----------------
        if (a.do_params) {
            bool params_changed = false;
#pragma unroll 1
            for (int l = 0; l < NP; ++l) {
                const int verdict = sm.s_in[set * kMaxNp + l];
                if (verdict == 0) continue;
                const double pl = sm.s_pl[set * kMaxNp + l], logu = sm.s_logu[set * kMaxNp + l];
                bool accept = false;
                if (verdict == 2) {
                    R pp[NP];
#pragma unroll
                    for (int k = 0; k < NP; ++k) pp[k] = (k == l) ? (R)pl : prm[k];
                    const typename Model::Prep pq = Model::prepare_move(prep, pp, a.dt, l);
                    const R* gc = cur ? sm.g1 : sm.g0;
                    R* ga = cur ? sm.g0 : sm.g1;
                    double part = 0.0;
                    {
                        R x0[D], x1[D], gp0[D], gp1[D], k0[NKA], k1[NKA];
                        lds_site<R, D>(sm.xs, 0, j, P, x0);
                        lds_site<R, D>(sm.xs, 1, j, P, x1);
#pragma unroll
                        for (int c = 0; c < NK; ++c) { k0[c] = sm.kg[c * P + j]; k1[c] = sm.kg[(NK + c) * P + j]; }
                        const R I0 = sm.Is[2 * j], I1 = sm.Is[2 * j + 1], I2 = sm.Is[2 * j + 2];
                        Model::template increment_k<(NK > 0), false>(x0, pp, pq, I0, I1, a.dt, gp0, k0, nullptr);
                        Model::template increment_k<(NK > 0), false>(x1, pp, pq, I1, I2, a.dt, gp1, k1, nullptr);
                        sts_site<R, D>(ga, 0, j, P, gp0);
                        sts_site<R, D>(ga, 1, j, P, gp1);
                        const int n0 = s_ext + 2 * j, n1 = n0 + 1;
                        const bool own0 = 2 * j < n_ext && n0 <= M - 1 && n0 >= s && n0 < e, own1 = 2 * j + 1 < n_ext && n1 <= M - 1 && n1 >= s && n1 < e;
                        R acc0 = R(0), acc1 = R(0);
#pragma unroll
                        for (int c = 0; c < D; ++c) {
                            const R d0 = x1[c] - x0[c], d1 = sm.xs[c * P + j + 1] - x1[c];
                            const R rn0 = d0 - gp0[c], ro0 = d0 - gc[c * P + j];
                            const R rn1 = d1 - gp1[c], ro1 = d1 - gc[(D + c) * P + j];
                            acc0 += R(0.5) * a.Rf[c] * (rn0 * rn0 - ro0 * ro0);
                            acc1 += R(0.5) * a.Rf[c] * (rn1 * rn1 - ro1 * ro1);
                        }
                        part = (own0 ? (double)acc0 : 0.0) + (own1 ? (double)acc1 : 0.0);
                    }
                    double dA = group_sum(part, sm.red, red_phase, grp, j);
                    if (G > 1) {   // all-gather of the chain's G partials as tagged packets; every group sums them in the same fixed order
                        const uint32_t tag = a.mc_tag0 + ar_count + 1u;
                        unsigned long long* base = a.mc_ar_words + ((size_t)(ar_count & 1u) * kMcMaxSlots + (size_t)cw * G) * kArSlotWords;
                        if (j == 0) ll_store_f64(base + (size_t)b * kArSlotWords, dA, tag);
                        const long long until = clock64() + (long long)a.ar_hold;
                        double mine = 0.0;
                        for (int jj = j; jj < G; jj += TG) {
                            if (jj == b) mine += dA;                    // own partial: no trip through L2
                            else {
                                while (clock64() < until) {}
                                mine += ll_wait_f64(base + (size_t)jj * kArSlotWords, tag, a.fault);
                            }
                        }
                        dA = group_sum(mine, sm.red, red_phase, grp, j);
                        ar_count += 1u;
                    }
                    accept = logu < -dA;
                    if (accept) cur ^= 1;
                    params_changed = params_changed || accept;
                }
#pragma unroll
                for (int k = 0; k < NP; ++k) prm[k] = (k == l && accept) ? (R)pl : prm[k];
                if (j == 0) { sm.s_pprop[l] += 1u; if (accept) sm.s_pacc[l] += 1u; }
            }
            if (params_changed) prep = Model::prepare(prm, a.dt);
        }

        // ---------------- A3: refresh the halos from the neighbour tiles (every h half-sweeps) ----------------
        if (G > 1 && a.do_states && i + 1 < a.n_sweeps && k_phase + 2 > h) {
            bar_group(grp);                          // every thread of the group is done with the tile's edge sites
            const uint32_t tag = a.mc_tag0 + hx_count + 1u;
            const size_t buf = (size_t)(hx_count & 1u);
            constexpr int WPV = sizeof(R) / 4;               // packets per value
            const int nwords = h * 2 * D * WPV;              // per direction
            const R* gc = cur ? sm.g1 : sm.g0;
            const uint32_t* xs32 = reinterpret_cast<const uint32_t*>(sm.xs);
            const uint32_t* gc32 = reinterpret_cast<const uint32_t*>(gc);
            for (int w = j; w < 2 * nwords; w += TG) {
                const int dir = w >= nwords ? 1 : 0, qq = w - dir * nwords;      // dir 0: to the left neighbour, 1: to the right
                if ((dir == 0 && b == 0) || (dir == 1 && b == G - 1)) continue;
                const int o = qq / (2 * D * WPV), rem = qq % (2 * D * WPV);
                const int which = rem / (D * WPV), cwd = rem % (D * WPV);
                const int nsite = dir == 0 ? s + o : e - h + o;
                const int widx = so<D>(nsite - s_ext, cwd / WPV, P) * WPV + cwd % WPV;
                uint32_t payload = 0;
                if (which == 0) payload = xs32[widx];
                else if (nsite <= M - 1) payload = gc32[widx];
                const int dst = mbox + (dir == 0 ? -1 : 1);
                const int dst_side = dir == 0 ? 1 : 0;           // my left neighbour receives "from its right"
                unsigned long long* box = a.mc_hx_words + (((size_t)dst * 2 + dst_side) * 2 + buf) * (size_t)kHaloWordsPerSide;
                ll_store(box + qq, payload, tag);
            }
            uint32_t* xd32 = reinterpret_cast<uint32_t*>(sm.xs);
            uint32_t* gd32 = reinterpret_cast<uint32_t*>(cur ? sm.g1 : sm.g0);
            for (int w = j; w < 2 * nwords; w += TG) {
                const int side = w >= nwords ? 1 : 0, qq = w - side * nwords;    // side 0: from the left neighbour, 1: from the right
                if ((side == 0 && b == 0) || (side == 1 && b == G - 1)) continue;
                const int o = qq / (2 * D * WPV), rem = qq % (2 * D * WPV);
                const int which = rem / (D * WPV), cwd = rem % (D * WPV);
                const int nsite = side == 0 ? s - h + o : e + o;
                const int widx = so<D>(nsite - s_ext, cwd / WPV, P) * WPV + cwd % WPV;
                const unsigned long long* box = a.mc_hx_words + (((size_t)mbox * 2 + side) * 2 + buf) * (size_t)kHaloWordsPerSide;
                const uint32_t payload = ll_wait(box + qq, tag, a.fault);
                if (which == 0) xd32[widx] = payload;
                else if (nsite <= M - 1) gd32[widx] = payload;
            }
            hx_count += 1u;
            k_phase = 0;
            bar_group(grp);
            if constexpr (NK > 0) { refresh_stage1(); bar_group(grp); }
        }

        // ---------------- A5: running moments and histograms (owned sites) ----------------
        if (acc_now) {
            if (!a.do_states) {       // otherwise the state moments were accumulated at decision time above
                for (int idx = (s - s_ext) * D + j; idx < (e - s_ext) * D; idx += TG) {
                    const int o = so<D>(idx / D, idx % D, P);
                    const double d = (double)sm.xs[o] - a.cx[(site0 + s_ext) * D + idx];
                    sm.S1[o] += d;
                    sm.S2[o] += d * d;
                }
            }
            if (b == 0 && j < NP) {
                double pv = 0.0;
#pragma unroll
                for (int k = 0; k < NP; ++k) pv = (k == j) ? (double)prm[k] : pv;
                const double d = pv - pcc;
                pS1 += d;
                pS2 += d * d;
                const unsigned long long rec = a.ptrace_n0 + n_rec;
                if (a.ptrace && rec < (unsigned long long)a.ptrace_cap) a.ptrace[((size_t)chain * a.ptrace_cap + rec) * NP + j] = (R)pv;
            }
            n_rec += 1ull;
            if (a.n_sel > 0) {
                for (int sel = j; sel < a.n_sel; sel += TG) {
                    const int site = a.hsite[sel], comp = a.hcomp[sel];
                    const bool mine = site < 0 ? (b == 0) : (site >= s && site < e);
                    if (mine) {
                        double v = 0.0;
                        if (site < 0) {
#pragma unroll
                            for (int k = 0; k < NP; ++k) v = (k == comp) ? (double)prm[k] : v;
                        } else v = (double)sm.xs[so<D>(site - s_ext, comp, P)];
                        unsigned long long* bins = a.hist + ((size_t)chain * a.n_sel + sel) * (size_t)(a.nbins + 2);
                        const double lo = a.hlo[sel], hi = a.hhi[sel];
                        int bin;
                        if (!(v >= lo)) bin = 0;
                        else if (v >= hi) bin = a.nbins + 1;
                        else {
                            long long qb = (long long)floor((v - lo) / a.hwidth[sel]);
                            if (qb >= a.nbins) qb = a.nbins - 1;
                            bin = 1 + (int)qb;
                        }
                        bins[bin] += 1ull;     // one owner thread per (chain, selection): no atomics needed
                    }
                }
                bar_group(grp);                // the next half-sweep overwrites x
            }
        }
    }

    // ---------------- write the tile back; A6 counters ----------------
    bar_group(grp);
    for (int idx = (s - s_ext) * D + j; idx < (e - s_ext) * D; idx += TG) gx[(size_t)s_ext * D + idx] = sm.xs[so<D>(idx / D, idx % D, P)];
    {
        R* gdst = cur ? gg1 : gg0;
        const R* gsrc = cur ? sm.g1 : sm.g0;
        const int hi_g = min(e, M);
        for (int idx = (s - s_ext) * D + j; idx < (hi_g - s_ext) * D; idx += TG) gdst[(size_t)s_ext * D + idx] = gsrc[so<D>(idx / D, idx % D, P)];
    }
    if (a.accum) {
        for (int idx = (s - s_ext) * D + j; idx < (e - s_ext) * D; idx += TG) {
            const size_t gi = (site0 + s_ext) * D + idx;
            const int o = so<D>(idx / D, idx % D, P);
            a.S1x[gi] = sm.S1[o]; a.S2x[gi] = sm.S2[o];
        }
        if (b == 0 && j < NP) {
            const size_t gi = (size_t)chain * NP + j;
            a.S1p[gi] = pS1; a.S2p[gi] = pS2;
        }
    }
    unsigned long long* cnt = a.counters + (size_t)chain * 2 * (D + NP);
    {
        unsigned int v = n_acc_state;
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, off);
        if ((j & 31) == 0 && v) {
#pragma unroll
            for (int c = 0; c < D; ++c) atomicAdd(cnt + c, (unsigned long long)v);      // a joint move counts for every component class
        }
    }
    if (j == 0) {
        const unsigned long long prop_u = a.do_states ? (unsigned long long)(e - s) * (unsigned long long)a.n_sweeps : 0ull;
        if (prop_u) {
#pragma unroll
            for (int c = 0; c < D; ++c) atomicAdd(cnt + (D + NP) + c, prop_u);
        }
        if (b == 0) {
#pragma unroll
            for (int l = 0; l < NP; ++l) {
                atomicAdd(cnt + D + l, (unsigned long long)sm.s_pacc[l]);
                atomicAdd(cnt + (D + NP) + D + l, (unsigned long long)sm.s_pprop[l]);
                a.p[(size_t)chain * NP + l] = prm[l];
            }
            a.cur[chain] = cur;
        }
    }
}

}  // namespace pimc

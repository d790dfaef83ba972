// Host side of libpimc: the C ABI declared in include/pimc.h (argument checks, workspace carving, launch
// configuration, absolute sweep counter).  All compute happens in the kernels of pimc_kernels.cuh; there
// is no CPU fallback.
#include "../../include/pimc.h"

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "pimc_kernels.cuh"
#include "pimc_tile_kernel.cuh"
#include "pimc_tilemc_kernel.cuh"

using namespace pimc;

// ---- translation-unit split (build time) ------------------------------------------------------------------------------
// This one source file is compiled five times (paper_1103_4887_b200/build.py, in parallel): PIMC_PART = 0 holds the C ABI
// and all host logic and instantiates NO sweep kernel; parts 1..4 each instantiate the kernels of one model family
// (1: HH tanh kinetics, 2: HH classic kinetics, 3: LINEAR fp64, 4: LINEAR fp32) behind one entry point, part_entry_<k>.
// PIMC_PART undefined = everything in one translation unit.
#ifndef PIMC_PART
#define PIMC_PART -1
#endif
#define PIMC_HAS_PART(k) (PIMC_PART == -1 || PIMC_PART == (k))

namespace pimc_shared {
#if PIMC_PART <= 0
thread_local std::string static_error;
#else
extern thread_local std::string static_error;
#endif
}  // namespace pimc_shared

namespace {

#define g_static_error pimc_shared::static_error

struct Carve {   // bump allocator over the caller's workspace; also used to size it
    char* base;
    size_t off = 0;
    explicit Carve(char* b) : base(b) {}
    template <typename T> T* take(size_t n) {
        off = (off + 255) & ~(size_t)255;
        T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
        off += n * sizeof(T);
        return p;
    }
};

struct Layout {
    void *x, *g0, *g1, *y, *I, *p, *kg;
    int* cur;
    double *lo, *hi, *cx, *S1x, *S2x, *cp, *S1p, *S2p;
    unsigned long long* counters;
    int *hsite, *hcomp;
    double *hlo, *hhi, *hwidth;
    unsigned long long* hist;
    unsigned long long *hs_flag, *ar_flag, *ar_epoch;
    double* ar_val;
    unsigned long long *hx_words, *hx_epoch, *ar_words;
    unsigned long long *mc_hx_words, *mc_ar_words;     // mailboxes of the many-chain tile-resident engine
    unsigned long long *st_words;                      // mailboxes of the sufficient-statistics exchange (trapezoid parameter moves)
    double *ws, *wpd;                 // tuned step sizes (C, M+1, D), (C, Np)
    unsigned int *nacc_s, *nacc_p;    // accepted changes since the last adjustment
    int* fault;
    size_t bytes;
};

constexpr int kMaxCtasPerChain = 1024;
constexpr size_t kMaxHistWords = 1u << 20;   // u64 counters reserved for histograms (all chains)

Layout carve(char* base, int D, int L, int M, int Np, int C, int dtype) {
    const size_t es = dtype == 64 ? 8 : 4;
    Carve c(base);
    Layout o{};
    const size_t nx = (size_t)C * (M + 1) * D, ng = (size_t)C * (M + 1) * D;   // caches: room for the trapezoid form's M + 1 entries
    o.x = c.take<char>(nx * es);
    o.g0 = c.take<char>(ng * es);
    o.g1 = c.take<char>(ng * es);
    o.kg = c.take<char>((size_t)C * (M + 1) * 3 * es);          // first-stage gate rates (NK <= 3 values per site)
    o.y = c.take<char>((size_t)C * (M + 1) * (L > 0 ? L : 1) * es);
    o.I = c.take<char>((size_t)C * (M + 1) * es);
    o.p = c.take<char>((size_t)C * Np * es);
    o.cur = c.take<int>(C);
    o.lo = c.take<double>((size_t)C * Np);
    o.hi = c.take<double>((size_t)C * Np);
    o.cx = c.take<double>(nx);
    o.S1x = c.take<double>(nx);
    o.S2x = c.take<double>(nx);
    o.cp = c.take<double>((size_t)C * Np);
    o.S1p = c.take<double>((size_t)C * Np);
    o.S2p = c.take<double>((size_t)C * Np);
    o.counters = c.take<unsigned long long>((size_t)C * 2 * (D + Np));
    o.hsite = c.take<int>(kMaxHistSel);
    o.hcomp = c.take<int>(kMaxHistSel);
    o.hlo = c.take<double>(kMaxHistSel);
    o.hhi = c.take<double>(kMaxHistSel);
    o.hwidth = c.take<double>(kMaxHistSel);
    o.hist = c.take<unsigned long long>(kMaxHistWords);
    o.hs_flag = c.take<unsigned long long>((size_t)C * kMaxCtasPerChain);
    o.ar_flag = c.take<unsigned long long>((size_t)C * 2 * kMaxCtasPerChain);
    o.ar_val = c.take<double>((size_t)C * 2 * kMaxCtasPerChain);
    o.ar_epoch = c.take<unsigned long long>(C);
    o.hx_epoch = c.take<unsigned long long>(C);
    o.hx_words = c.take<unsigned long long>((size_t)kTileMaxCtas * 2 * 2 * kHaloWordsPerSide);
    o.ar_words = c.take<unsigned long long>((size_t)2 * kTileMaxCtas * kArSlotWords);
    o.mc_hx_words = c.take<unsigned long long>((size_t)kMcMaxSlots * 2 * 2 * kHaloWordsPerSide);
    o.mc_ar_words = c.take<unsigned long long>((size_t)2 * kMcMaxSlots * kArSlotWords);
    o.st_words = c.take<unsigned long long>((size_t)2 * kTileMaxCtas * 2 * kStatSlots * 2);
    o.ws = c.take<double>(nx);
    o.wpd = c.take<double>((size_t)C * Np);
    o.nacc_s = c.take<unsigned int>(nx);
    o.nacc_p = c.take<unsigned int>((size_t)C * Np);
    o.fault = c.take<int>(4);
    o.bytes = (c.off + 255) & ~(size_t)255;
    return o;
}

bool shape_ok(int model, int D, int L, int M, int C, int dtype, int* why) {
    *why = PIMC_EINVAL;
    if (!(model == PIMC_MODEL_LINEAR || model == PIMC_MODEL_HH || model == PIMC_MODEL_HH_CLASSIC)) return false;
    if (D < 1 || L < 0 || L > D || M < 1 || C < 1 || !(dtype == 64 || dtype == 32)) return false;
    *why = PIMC_EUNSUPPORTED;
    if (model != PIMC_MODEL_LINEAR && D != 4) return false;
    if (model == PIMC_MODEL_LINEAR && D > 4) return false;
    if ((long long)C * ((long long)M + 1) > (1ll << 31)) return false;
    return true;
}

}  // namespace

struct pimc_handle {
    int model, D, L, M, Np, C, dtype;
    double dt, Rm, Rf[kMaxD];
    cudaStream_t stream;
    Layout lay;
    double wx[kMaxD], wp[kMaxNp];
    int kind = 0;
    int disc = PIMC_DISC_RK4MAP;
    int update_mode = PIMC_UPDATE_JOINT;
    double beta0 = 1.0; unsigned long long n_cool = 0, t_anneal = 0;
    bool site_widths = false;         // per-(site, component) step sizes in use (step-size tuning was switched on since the last set_proposal)
    int tune = 0; unsigned long long tune_skip = 1, t_tune = 0; double f_acc = 0.23, alpha = 0.02;
    bool have_data = false, have_path = false, have_prop = false, have_I = false;
    int accum = 0;
    unsigned long long n_skip = 1, t_enable = 0, n_samples = 0, t = 0;
    int n_sel = 0, nbins = 0;
    void *tr_dA = nullptr, *tr_xprop = nullptr, *tr_dAp = nullptr, *tr_pprop = nullptr;
    unsigned char *tr_acc = nullptr, *tr_accp = nullptr;
    int G_user = 0, T_user = 0, engine_user = PIMC_ENGINE_AUTO, halo_user = -1;
    unsigned long long hs_base = 0, launches = 0;
    int ar_hold = 450;                // pimc_set_exchange
    unsigned long long mc_tag = 1;    // next unused tag of the many-chain engine's mailboxes (every launch takes a private range)
    bool kg_valid = false;            // the global first-stage gate-rate array matches the path (GLOBAL engine keeps it current, TILE does not)
    void* ptrace = nullptr; long long ptrace_cap = 0;      // pimc_param_trace
    double* resid_acc = nullptr;                           // pimc_set_residual_stats
    int sm_count = 0;
    std::string err;
};

namespace {

// SM count of the current device (grid sizing of the helper kernels); 148 on B200, never assumed
int sm_count_now() {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) return 1;
    return sms;
}
// caller-provided device arrays must be 32-byte aligned (SURVEY.md §8(b) conventions: vectorised loads)
bool aligned32(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 31u) == 0; }

int fail(pimc_handle* h, int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (h) h->err = buf;                 // the message of the LATEST failure (pimc_last_error)
    else g_static_error = buf;
    return code;
}
#define PIMC_CUDA(h, call)                                                                        \
    do {                                                                                          \
        cudaError_t e_ = (call);                                                                  \
        if (e_ != cudaSuccess) return fail(h, PIMC_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
    } while (0)

// ---- model / dtype dispatch --------------------------------------------------------------------------
// The four operations that need a model's kernels, behind one entry point per model family (see the split above).
enum { OP_REBUILD = 0, OP_SWEEP = 1, OP_SHAPE = 2, OP_STEP = 3 };
}  // namespace
namespace pimc_shared {
struct LaunchShape { int G, T, tile; bool cooperative; int engine, h; size_t smem; int cpw, waves; };   // cpw: chains per wave (TILE_MC)
struct OpArgs {
    int op;
    pimc_handle* h;
    long long n_sweeps; unsigned long long seed; int do_states, do_params;     // OP_SWEEP
    LaunchShape* ls;                                                           // OP_SHAPE
    const void *x, *p, *I0, *I1; double dt; unsigned long long n; void* g; void* stream;   // OP_STEP
};
int part_entry_1(int model, int D, int dtype, const OpArgs& o);   // HH, tanh kinetics
int part_entry_2(int model, int D, int dtype, const OpArgs& o);   // HH, classic kinetics
int part_entry_3(int model, int D, int dtype, const OpArgs& o);   // LINEAR, fp64
int part_entry_4(int model, int D, int dtype, const OpArgs& o);   // LINEAR, fp32
}  // namespace pimc_shared
using pimc_shared::LaunchShape;
using pimc_shared::OpArgs;
namespace {
int dispatch_op(int model, int D, int dtype, const OpArgs& o) {
    if (model == PIMC_MODEL_HH) return pimc_shared::part_entry_1(model, D, dtype, o);
    if (model == PIMC_MODEL_HH_CLASSIC) return pimc_shared::part_entry_2(model, D, dtype, o);
    if (model == PIMC_MODEL_LINEAR) return dtype == 64 ? pimc_shared::part_entry_3(model, D, dtype, o) : pimc_shared::part_entry_4(model, D, dtype, o);
    return PIMC_EUNSUPPORTED;
}

// Choose CTAs per chain, threads per CTA and the tile length (even).
template <class Model, typename R> int choose_shape_global(pimc_handle* h, LaunchShape* out) {
    int T = h->T_user;
    int G = h->G_user;
    const int sites = h->M + 1;
    int per_sm = 0;
    if (G == 0) {
        // many chains: one CTA per chain, no inter-CTA traffic.  few chains: spread each over the SMs.
        if (h->C >= h->sm_count / 2) G = 1;
        else {
            if (T == 0) T = 128;
            PIMC_CUDA(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, sweep_kernel<Model, R, false>, T, 0));
            const int cap = per_sm > 0 ? h->sm_count : 0;    // one CTA per SM: the FP64 pipe is the shared resource
            G = (sites + 2 * T - 1) / (2 * T);
            if (G > cap / h->C) G = cap / h->C;
            if (G < 1) G = 1;
        }
    }
    if (T == 0) T = (G == 1) ? kMaxThreads : 128;
    if (T % 32 != 0 || T < 32 || T > kMaxThreads) return fail(h, PIMC_EINVAL, "threads_per_cta must be a multiple of 32 in [32,%d]", kMaxThreads);
    if (G > kMaxCtasPerChain) return fail(h, PIMC_EINVAL, "ctas_per_chain > %d", kMaxCtasPerChain);
    int tile = (sites + G - 1) / G;
    tile += tile & 1;
    G = (sites + tile - 1) / tile;     // drop empty tiles
    out->G = G; out->T = T; out->tile = tile; out->cooperative = G > 1;
    out->engine = PIMC_ENGINE_GLOBAL; out->h = 0; out->smem = 0;
    if (G > 1) {
        PIMC_CUDA(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, sweep_kernel<Model, R, false>, T, 0));
        if ((long long)G * h->C > (long long)per_sm * h->sm_count)
            return fail(h, PIMC_EINVAL, "grid of %d CTAs is not co-resident (capacity %d)", G * h->C, per_sm * h->sm_count);
    }
    return PIMC_OK;
}

// Tile-resident engine: G tiles per chain, each tile plus 2 h halo sites fits the 2 TC = T threads of its CTA
// (one (even, odd) site pair per compute thread).  Returns PIMC_EUNSUPPORTED (without touching the error string)
// when the problem does not fit, so that the automatic choice can fall back to the global-memory engine.
template <class Model, typename R> int choose_shape_tile(pimc_handle* h, LaunchShape* out, bool quiet) {
    const int sites = h->M + 1;
    const int cap_ctas = std::min(h->sm_count, kTileMaxCtas);      // one CTA per SM: the FP64 pipe is the shared resource
    auto no = [&](const char* why) { return quiet ? (int)PIMC_EUNSUPPORTED : fail(h, PIMC_EUNSUPPORTED, "tile engine: %s", why); };
    if (h->L != 1) return no("the tile engine is compiled for one observed component (L = 1)");
    if (h->C > cap_ctas) return no("more chains than co-resident CTAs");
    int T = h->T_user, G = h->G_user;
    // the 512-thread instantiation exists for the RK4-map, joint-update kernel only (build time); the others stop at 256
    const int Tcap = (h->disc != PIMC_DISC_RK4MAP || h->update_mode != PIMC_UPDATE_JOINT) ? 256 : 512;
    if (T != 0 && (T % 64 != 0 || T > Tcap)) return no("threads_per_cta must be a multiple of 64, at most 512 (256 for the trapezoid rule or component-wise updates)");
    const int Tmax = T ? T : Tcap;
    const int h_want = h->halo_user >= 0 ? h->halo_user : kTileHaloMax;
    if (G == 0) {
        if (sites <= (T ? T : 256)) G = 1;                          // whole chain in one CTA: no hand-off at all
        else {
            G = cap_ctas / h->C;                                    // spread each chain over as many SMs as there are
            const int min_tile = 32;
            if (G > (sites + min_tile - 1) / min_tile) G = (sites + min_tile - 1) / min_tile;
            if (G < 1) G = 1;
        }
    }
    if ((long long)G * h->C > cap_ctas && G > 1) return no("grid would not be co-resident");
    // In a parameter move every CTA polls the G partial sums of its chain, one mailbox line per thread: with more tiles than
    // threads some threads wait for two lines in turn, a second trip through L2 per move (measured at M = 8000: 23.0 us per sweep
    // with 143 tiles of 128 threads, 15.4 with 122).  The automatic choice therefore keeps G <= T (second pass of this loop).
    const bool auto_shape = h->G_user == 0 && h->T_user == 0;
    int tile = 0, hh = 0;
    for (int pass = 0; pass < 2; ++pass) {
        tile = (sites + G - 1) / G;
        tile += tile & 1;
        for (;;) {                                                  // the last tile must not be shorter than 2 sites
            G = (sites + tile - 1) / tile;
            const int last = sites - (G - 1) * tile;
            if (G == 1 || last >= 2) break;
            tile += 2;
        }
        hh = 0;
        if (G > 1) {
            const int last = sites - (G - 1) * tile;
            hh = std::min(h_want, kTileHaloMax) & ~1;
            hh = std::min(hh, last & ~1);
            hh = std::min(hh, tile & ~1);
            hh = std::min(hh, ((Tmax - tile) / 2) & ~1);
            if (hh < 2) return no("tile plus halos does not fit the CTA");
        }
        int Tneed = std::max(64, (tile + 2 * hh + 63) / 64 * 64);
        // 192 threads are 3 compute + 3 producer warps on 4 schedulers; 4 + 4 run 3-5 % faster (M = 16384: 20.3 -> 19.5 us per sweep)
        if (auto_shape && Tneed == 192 && Tcap >= 256) Tneed = 256;
        if (pass == 0 && auto_shape && G > Tneed && Tneed <= Tcap) { G = Tneed; continue; }
        if (T == 0) T = Tneed;
        break;
    }
    if (tile + 2 * hh > T || T > Tcap) return no("tile plus halos does not fit the CTA");
    out->G = G; out->T = T; out->tile = tile; out->cooperative = G > 1; out->engine = PIMC_ENGINE_TILE; out->h = hh;
    out->smem = tile_smem_bytes<R>(T, h->D, h->L, h->disc == PIMC_DISC_TRAPEZOID ? 0 : Model::NK, h->update_mode == PIMC_UPDATE_COMPONENTWISE ? h->D : 1,
                                   h->disc == PIMC_DISC_TRAPEZOID && Model::NTH > 0);
    if (out->smem > 227 * 1024) return no("shared memory");
    return PIMC_OK;
}

// Many-chain tile-resident engine (pimc_tilemc_kernel.cuh): every CTA hosts NGRP groups of 128 threads, each with one
// (chain, tile) pair of at most 256 sites incl. halos; chains that do not fit at once run in waves of `cpw` chains.
template <class Model, typename R> int choose_shape_mc(pimc_handle* h, LaunchShape* out, bool quiet) {
    auto no = [&](const char* why) { return quiet ? (int)PIMC_EUNSUPPORTED : fail(h, PIMC_EUNSUPPORTED, "many-chain tile engine: %s", why); };
    if constexpr (!Model::kTileMc) return no("not compiled for this model");
    else {
        if (h->L != 1) return no("compiled for one observed component (L = 1)");
        if (h->disc != PIMC_DISC_RK4MAP || h->update_mode != PIMC_UPDATE_JOINT) return no("RK4-map discretisation with joint updates only");
        if (h->site_widths) return no("per-site step sizes (step-size tuning) are not supported");
        if (h->tr_dA || h->tr_acc || h->tr_xprop || h->tr_dAp || h->tr_accp || h->tr_pprop) return no("the debug trace is not supported");
        if (h->n_cool != 0 && h->t < h->t_anneal + h->n_cool) return no("annealing is not supported");
        const int sites = h->M + 1;
        int T = h->T_user ? h->T_user : 4 * kMcGroup;
        if (T != 2 * kMcGroup && T != 3 * kMcGroup && T != 4 * kMcGroup) return no("threads_per_cta must be 256, 384 or 512 (2, 3 or 4 groups of 128)");
        const int NG = T / kMcGroup;
        int hh = h->halo_user >= 0 ? h->halo_user : 8, G = h->G_user, tile = 0;
        if (G == 0 && sites <= kMcTileMax) G = 1;
        if (G == 1) { tile = sites + (sites & 1); hh = 0; }
        else {
            if (hh < 2) return no("halo depth must be at least 2 with more than one tile per chain");
            const int cap = kMcTileMax - 2 * hh;
            if (G == 0) G = (sites + cap - 1) / cap;
            tile = (sites + G - 1) / G;
            tile += tile & 1;
            for (;;) {                                                  // the last tile must hold at least the h sites it sends
                G = (sites + tile - 1) / tile;
                const int last = sites - (G - 1) * tile;
                if (G == 1 || last >= hh) break;
                tile += 2;
            }
            if (G == 1) hh = 0;
        }
        if (tile + 2 * hh > kMcTileMax) return no("tile plus halos exceeds 256 sites");
        const int slots = std::min(h->sm_count * NG, kMcMaxSlots);
        int cpw = std::min(slots / G, h->C);
        if (cpw < 1) return no("a chain does not fit the co-resident groups");
        const int waves = (h->C + cpw - 1) / cpw;
        cpw = (h->C + waves - 1) / waves;                               // even waves
        out->G = G; out->T = T; out->tile = tile; out->cooperative = true; out->engine = PIMC_ENGINE_TILE_MC; out->h = hh;
        out->smem = (size_t)NG * mc_group_bytes<R>(h->D, Model::NK);
        out->cpw = cpw; out->waves = waves;
        if (out->smem > 227 * 1024) return no("shared memory");
        return PIMC_OK;
    }
}

// AUTO: the tile-resident engine when the problem fits it; several chains that do not: the many-chain tile-resident engine;
// everything else: the global-memory engine.
template <class Model, typename R> int choose_shape(pimc_handle* h, LaunchShape* out) {
    out->cpw = h->C; out->waves = 1;
    if (h->engine_user == PIMC_ENGINE_GLOBAL) return choose_shape_global<Model, R>(h, out);
    if (h->engine_user == PIMC_ENGINE_TILE) return choose_shape_tile<Model, R>(h, out, false);
    if (h->engine_user == PIMC_ENGINE_TILE_MC) return choose_shape_mc<Model, R>(h, out, false);
    if (choose_shape_tile<Model, R>(h, out, true) == PIMC_OK) return PIMC_OK;
    if (h->C >= 2 && h->G_user == 0 && h->T_user == 0 && choose_shape_mc<Model, R>(h, out, true) == PIMC_OK) return PIMC_OK;
    out->cpw = h->C; out->waves = 1;
    return choose_shape_global<Model, R>(h, out);
}

template <class Model, typename R> int rebuild_cache(pimc_handle* h) {
    const size_t total = (size_t)h->C * (h->M + 1);
    const int threads = 128;
    const int blocks = (int)std::min<size_t>((total + threads - 1) / threads, (size_t)h->sm_count * 16);
    // after a rebuild, buffer 0 is current
    build_cache_kernel<Model, R><<<blocks, threads, 0, h->stream>>>((const R*)h->lay.x, h->have_I ? (const R*)h->lay.I : nullptr,
                                                                     (const R*)h->lay.p, (R*)h->lay.g0, h->M, h->C, (R)h->dt, h->disc, (R*)h->lay.kg);
    h->launches++;
    PIMC_CUDA(h, cudaGetLastError());
    PIMC_CUDA(h, cudaMemsetAsync(h->lay.cur, 0, sizeof(int) * h->C, h->stream));
    h->kg_valid = h->disc == PIMC_DISC_RK4MAP;
    return PIMC_OK;
}

int rebuild(pimc_handle* h) {
    OpArgs o{}; o.op = OP_REBUILD; o.h = h;
    return dispatch_op(h->model, h->D, h->dtype, o);
}

template <class Model, typename R> int run_sweeps_once(pimc_handle* h, long long n_sweeps, unsigned long long seed, int do_states, int do_params) {
    LaunchShape ls;
    int rc = choose_shape<Model, R>(h, &ls);
    if (rc != PIMC_OK) return rc;
    SweepArgs<R> a{};
    a.M = h->M; a.L = h->L; a.n_chains = h->C; a.G = ls.G; a.tile = ls.tile; a.kind = h->kind;
    a.update_mode = h->update_mode;
    a.ws = h->site_widths ? h->lay.ws : nullptr; a.nacc_s = h->lay.nacc_s; a.wpd = h->lay.wpd; a.nacc_p = h->lay.nacc_p;
    a.tune = h->site_widths ? h->tune : 0; a.tune_skip = h->tune_skip; a.t_tune = h->t_tune; a.f_acc = h->f_acc; a.alpha = h->alpha;
    a.ln_beta0 = std::log(h->beta0); a.n_cool = h->n_cool; a.t_anneal = h->t_anneal;
    a.disc = h->disc; a.nc = h->disc == PIMC_DISC_TRAPEZOID ? h->M + 1 : h->M;
    a.dt = (R)h->dt; a.Rm = (R)h->Rm;
    for (int c = 0; c < h->D; ++c) { a.Rf[c] = (R)h->Rf[c]; a.wx[c] = (R)h->wx[c]; }
    for (int l = 0; l < h->Np; ++l) a.wp[l] = h->wp[l];
    a.x = (R*)h->lay.x; a.g[0] = (R*)h->lay.g0; a.g[1] = (R*)h->lay.g1; a.kg = (R*)h->lay.kg;
    a.y = (const R*)h->lay.y; a.I = h->have_I ? (const R*)h->lay.I : nullptr;
    a.p = (R*)h->lay.p; a.cur = h->lay.cur; a.lo = h->lay.lo; a.hi = h->lay.hi;
    a.accum = h->accum; a.n_skip = h->n_skip; a.t_enable = h->t_enable; a.skip0 = h->accum ? (h->t - h->t_enable) % h->n_skip : 0ull;
    a.cx = h->lay.cx; a.S1x = h->lay.S1x; a.S2x = h->lay.S2x; a.cp = h->lay.cp; a.S1p = h->lay.S1p; a.S2p = h->lay.S2p;
    a.counters = h->lay.counters;
    a.n_sel = h->n_sel; a.nbins = h->nbins;
    a.hsite = h->lay.hsite; a.hcomp = h->lay.hcomp; a.hlo = h->lay.hlo; a.hhi = h->lay.hhi; a.hwidth = h->lay.hwidth; a.hist = h->lay.hist;
    a.tr_dA = (R*)h->tr_dA; a.tr_acc = h->tr_acc; a.tr_xprop = (R*)h->tr_xprop;
    a.tr_dAp = (R*)h->tr_dAp; a.tr_accp = h->tr_accp; a.tr_pprop = (R*)h->tr_pprop;
    a.t0 = h->t; a.seed = seed; a.n_sweeps = n_sweeps; a.do_states = do_states; a.do_params = do_params;
    a.hs_flag = h->lay.hs_flag; a.ar_val = h->lay.ar_val; a.ar_flag = h->lay.ar_flag; a.ar_epoch = h->lay.ar_epoch;
    a.hs_base = h->hs_base;
    a.h = ls.h; a.hx_words = h->lay.hx_words; a.hx_epoch = h->lay.hx_epoch; a.ar_words = h->lay.ar_words; a.fault = h->lay.fault; a.ar_hold = h->ar_hold; a.st_words = h->lay.st_words;
    a.ptrace = (R*)h->ptrace; a.ptrace_cap = h->ptrace_cap; a.ptrace_n0 = h->n_samples;
    a.mc_hx_words = h->lay.mc_hx_words; a.mc_ar_words = h->lay.mc_ar_words; a.mc_chain0 = 0; a.mc_nchains = h->C; a.mc_tag0 = 0;

    const dim3 grid((unsigned)(ls.G * h->C)), block((unsigned)ls.T);
    const bool trap = h->disc == PIMC_DISC_TRAPEZOID;
    const void* fn = ls.G == 1 ? (const void*)sweep_kernel<Model, R, true> : (const void*)sweep_kernel<Model, R, false>;
    if (ls.engine == PIMC_ENGINE_TILE) {
        const bool comp = h->update_mode == PIMC_UPDATE_COMPONENTWISE;
        // the stage-1 cache is only worth keeping if this launch moves a parameter (and the model has one: NK > 0)
        bool kg = false;
        if constexpr (Model::NK > 0) {
            if (do_params && !trap) {
                kg = h->site_widths;                                   // tuned parameter step sizes live on the device
                for (int l = 0; l < h->Np; ++l) kg = kg || h->wp[l] > 0.0;
            }
        }
        // the general variant (template flag TR): debug trace requested, or a sweep of this launch has the annealing multiplier below 1
        const bool tr = h->tr_dA || h->tr_acc || h->tr_xprop || h->tr_dAp || h->tr_accp || h->tr_pprop ||
                        (h->n_cool != 0 && h->t < h->t_anneal + h->n_cool && h->t + (unsigned long long)n_sweeps > h->t_anneal) ||
                        (h->site_widths && h->tune);
        constexpr bool HK = Model::NK > 0;
        const int sel = (ls.T <= 256 ? 0 : 4) + (trap ? 2 : 0) + (comp ? 1 : 0);
#define PIMC_TILE(MAXT_, TRAP_, COMP_, KG_) \
    (tr ? (const void*)tile_sweep_kernel<Model, R, MAXT_, TRAP_, COMP_, KG_, true> : (const void*)tile_sweep_kernel<Model, R, MAXT_, TRAP_, COMP_, KG_, false>)
        switch (sel) {
            case 0: fn = kg ? PIMC_TILE(256, false, false, HK) : PIMC_TILE(256, false, false, false); break;
            case 1: fn = kg ? PIMC_TILE(256, false, true, HK) : PIMC_TILE(256, false, true, false); break;
            case 2: fn = PIMC_TILE(256, true, false, false); break;
            case 3: fn = PIMC_TILE(256, true, true, false); break;
            case 4: fn = kg ? PIMC_TILE(512, false, false, HK) : PIMC_TILE(512, false, false, false); break;
            default: return fail(h, PIMC_EUNSUPPORTED, "no 512-thread tile kernel for this discretisation / update mode");   // choose_shape_tile never offers it
        }
#undef PIMC_TILE
    }
    if constexpr (Model::NK > 0) {
        if (ls.engine == PIMC_ENGINE_GLOBAL && !trap && !h->kg_valid) {      // the previous launches ran tile-resident: refresh the stage-1 rates
            const size_t total = (size_t)h->C * h->M;
            const int threads = 128;
            const int blocks = (int)std::min<size_t>((total + threads - 1) / threads, (size_t)h->sm_count * 16);
            build_stage1_kernel<Model, R><<<blocks, threads, 0, h->stream>>>((const R*)h->lay.x, h->M, h->C, (R*)h->lay.kg);
            h->launches++;
            PIMC_CUDA(h, cudaGetLastError());
            h->kg_valid = true;
        }
        if (ls.engine != PIMC_ENGINE_GLOBAL && do_states) h->kg_valid = false;
    }
    if constexpr (Model::kTileMc) {
        if (ls.engine == PIMC_ENGINE_TILE_MC) {
            // one launch per wave of ls.cpw chains, each running all n_sweeps on its chains; every launch gets a private tag range
            const int NG = ls.T / kMcGroup;
            fn = NG == 4 ? (const void*)tilemc_sweep_kernel<Model, R, 4> : NG == 3 ? (const void*)tilemc_sweep_kernel<Model, R, 3> : (const void*)tilemc_sweep_kernel<Model, R, 2>;
            PIMC_CUDA(h, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ls.smem));
            const unsigned long long span = (unsigned long long)n_sweeps * (unsigned long long)(Model::NP + 1) + 4ull;
            if (span >= (1ull << 31)) return fail(h, PIMC_EINVAL, "too many sweeps for one call of the many-chain tile engine");
            for (int w = 0; w < ls.waves; ++w) {
                if ((h->mc_tag & 0xFFFFFFFFull) + span >= (1ull << 32)) {   // the 32-bit tags would wrap inside this launch: start a new epoch
                    PIMC_CUDA(h, cudaMemsetAsync(h->lay.mc_hx_words, 0, sizeof(unsigned long long) * (size_t)kMcMaxSlots * 2 * 2 * kHaloWordsPerSide, h->stream));
                    PIMC_CUDA(h, cudaMemsetAsync(h->lay.mc_ar_words, 0, sizeof(unsigned long long) * (size_t)2 * kMcMaxSlots * kArSlotWords, h->stream));
                    h->mc_tag = (h->mc_tag | 0xFFFFFFFFull) + 2ull;          // low word = 1: tag 0 (fresh memory) is never awaited
                }
                a.mc_chain0 = w * ls.cpw;
                a.mc_nchains = std::min(ls.cpw, h->C - a.mc_chain0);
                a.mc_tag0 = (unsigned int)(h->mc_tag & 0xFFFFFFFFull);
                h->mc_tag += span;
                const int groups = a.mc_nchains * ls.G;
                const dim3 mc_grid((unsigned)std::min(h->sm_count, groups));
                void* mc_params[] = {&a};
                PIMC_CUDA(h, cudaLaunchCooperativeKernel(fn, mc_grid, block, mc_params, ls.smem, h->stream));
                h->launches++;
            }
        }
    }
    if (ls.engine == PIMC_ENGINE_TILE_MC) {
        if constexpr (!Model::kTileMc) return fail(h, PIMC_EUNSUPPORTED, "many-chain tile engine: not compiled for this model");
    } else {
    if (ls.smem > 48 * 1024) PIMC_CUDA(h, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ls.smem));
    void* params[] = {&a};
    if (ls.cooperative) PIMC_CUDA(h, cudaLaunchCooperativeKernel(fn, grid, block, params, ls.smem, h->stream));
    else PIMC_CUDA(h, cudaLaunchKernel(fn, grid, block, params, ls.smem, h->stream));
    h->launches++;
    }
    if (do_states && ls.engine == PIMC_ENGINE_GLOBAL) h->hs_base += 2ull * (unsigned long long)n_sweeps;
    if (h->accum) {   // host bookkeeping of the sample count: sweeps t in [t0, t0+n) with (t - t_enable) % n_skip == 0
        const unsigned long long first = h->t - h->t_enable, last = first + (unsigned long long)n_sweeps;   // [first, last)
        const unsigned long long k = h->n_skip;
        h->n_samples += (last + k - 1) / k - (first + k - 1) / k;
    }
    h->t += (unsigned long long)n_sweeps;
    return PIMC_OK;
}

// While the step sizes are being tuned the tile-resident engine cannot adjust them inside a launch (its producer
// warps have drawn the next sweep's proposals already, and the halo copies of a site do not see all of its decisions), so the
// launcher ends every launch at an adjustment sweep -- (t - t_tune + 1) % tune_skip == 0 -- and runs tune_adjust_kernel on the
// counters the owners kept.  The global-memory engine adjusts inside its kernel; both give the oracle's step sizes bit for bit.
template <typename R> int accumulate_residuals(pimc_handle* h) {
    const size_t total = (size_t)h->C * (h->M + 1);
    const int threads = 256;
    const int blocks = (int)std::min<size_t>((total + threads - 1) / threads, (size_t)h->sm_count * 8);
    residual_kernel<R><<<blocks, threads, 0, h->stream>>>((const R*)h->lay.x, (const R*)h->lay.g0, (const R*)h->lay.g1, h->lay.cur, (const R*)h->lay.y,
                                                          h->M, h->D, h->L, h->disc == PIMC_DISC_TRAPEZOID ? h->M + 1 : h->M, h->disc, h->C,
                                                          nullptr, nullptr, h->resid_acc);
    h->launches++;
    PIMC_CUDA(h, cudaGetLastError());
    return PIMC_OK;
}

// A pimc_sweep call is ONE launch unless something has to happen between two sweeps on the host's side of the kernel:
//  * step-size tuning on the tile-resident engine: every launch ends at an adjustment sweep, tune_adjust_kernel runs in between;
//  * residual statistics (pimc_set_residual_stats): every launch ends at an accumulated sweep, residual_kernel adds that path's
//    eps_n, delta_n to the running sums (a diagnostic: one extra launch per sample, nothing added to the sweep kernels).
template <class Model, typename R> int run_sweeps(pimc_handle* h, long long n_sweeps, unsigned long long seed, int do_states, int do_params) {
    const bool want_tune = h->site_widths && h->tune, want_res = h->resid_acc != nullptr && h->accum;
    if (!(want_tune || want_res) || n_sweeps <= 0) return run_sweeps_once<Model, R>(h, n_sweeps, seed, do_states, do_params);
    LaunchShape ls;
    int rc = choose_shape<Model, R>(h, &ls);
    if (rc != PIMC_OK) return rc;
    const bool split_tune = want_tune && ls.engine == PIMC_ENGINE_TILE;
    if (!split_tune && !want_res) return run_sweeps_once<Model, R>(h, n_sweeps, seed, do_states, do_params);
    long long left = n_sweeps;
    while (left > 0) {
        unsigned long long to_adjust = ~0ull, to_acc = ~0ull;
        if (split_tune) to_adjust = h->tune_skip - (h->t - h->t_tune) % h->tune_skip;   // up to and including the adjustment sweep
        if (want_res) {                                                                // up to and including the next accumulated sweep
            const unsigned long long r = (h->t - h->t_enable) % h->n_skip;
            to_acc = (r == 0 ? 0ull : h->n_skip - r) + 1ull;
        }
        const unsigned long long stop = std::min(to_adjust, to_acc);
        const long long n = (unsigned long long)left < stop ? left : (long long)stop;
        rc = run_sweeps_once<Model, R>(h, n, seed, do_states, do_params);
        if (rc != PIMC_OK) return rc;
        if (split_tune && (unsigned long long)n == to_adjust) {
            const size_t nx = (size_t)h->C * (h->M + 1) * h->D, np = (size_t)h->C * h->Np;
            const int threads = 256;
            const int blocks = (int)std::min<size_t>((nx + np + threads - 1) / threads, (size_t)h->sm_count * 8);
            tune_adjust_kernel<<<blocks, threads, 0, h->stream>>>(h->lay.ws, h->lay.nacc_s, nx, h->lay.wpd, h->lay.nacc_p, np,
                                                                   (double)h->tune_skip, h->f_acc, h->alpha);
            PIMC_CUDA(h, cudaGetLastError());
            h->launches++;
        }
        if (want_res && (unsigned long long)n == to_acc) {
            rc = accumulate_residuals<R>(h);
            if (rc != PIMC_OK) return rc;
        }
        left -= n;
    }
    return PIMC_OK;
}

template <class Model, typename R> int run_op(const OpArgs& o) {
    switch (o.op) {
        case OP_REBUILD: return rebuild_cache<Model, R>(o.h);
        case OP_SWEEP: return run_sweeps<Model, R>(o.h, o.n_sweeps, o.seed, o.do_states, o.do_params);
        case OP_SHAPE: return choose_shape<Model, R>(o.h, o.ls);
        case OP_STEP: {
            const int threads = 128;
            const int blocks = (int)std::min<unsigned long long>((o.n + threads - 1) / threads, (unsigned long long)sm_count_now() * 16);
            step_selftest_kernel<Model, R><<<blocks, threads, 0, (cudaStream_t)o.stream>>>((const R*)o.x, (const R*)o.p, (const R*)o.I0, (const R*)o.I1,
                                                                                         (R)o.dt, o.n, (R*)o.g);
            PIMC_CUDA(nullptr, cudaGetLastError());
            return PIMC_OK;
        }
    }
    return PIMC_EINVAL;
}
}  // namespace

// ---- the model families: each entry point is compiled in exactly one translation unit --------------------------------
namespace pimc_shared {
#if PIMC_HAS_PART(1)
int part_entry_1(int, int, int dtype, const OpArgs& o) { return dtype == 64 ? run_op<HHModel<double>, double>(o) : run_op<HHModel<float>, float>(o); }
#endif
#if PIMC_HAS_PART(2)
int part_entry_2(int, int, int dtype, const OpArgs& o) { return dtype == 64 ? run_op<HHClassicModel<double>, double>(o) : run_op<HHClassicModel<float>, float>(o); }
#endif
#if PIMC_HAS_PART(3)
int part_entry_3(int, int D, int, const OpArgs& o) {
    switch (D) {
        case 1: return run_op<LinearModel<double, 1>, double>(o);
        case 2: return run_op<LinearModel<double, 2>, double>(o);
        case 3: return run_op<LinearModel<double, 3>, double>(o);
        case 4: return run_op<LinearModel<double, 4>, double>(o);
    }
    return PIMC_EUNSUPPORTED;
}
#endif
#if PIMC_HAS_PART(4)
int part_entry_4(int, int D, int, const OpArgs& o) {
    switch (D) {
        case 1: return run_op<LinearModel<float, 1>, float>(o);
        case 2: return run_op<LinearModel<float, 2>, float>(o);
        case 3: return run_op<LinearModel<float, 3>, float>(o);
        case 4: return run_op<LinearModel<float, 4>, float>(o);
    }
    return PIMC_EUNSUPPORTED;
}
#endif
}  // namespace pimc_shared

#if PIMC_PART <= 0      // the C ABI and its host-side helpers: part 0 (or the single translation unit) only
namespace {

int sweep_common(pimc_handle* h, long long n_sweeps, unsigned long long seed, int do_states, int do_params) {
    if (!h) return PIMC_EINVAL;
    if (n_sweeps < 0) return fail(h, PIMC_EINVAL, "n_sweeps < 0");
    if (!h->have_data || !h->have_path || !h->have_prop) return fail(h, PIMC_ESTATE, "pimc_sweep before set_data / set_path / set_proposal");
    if (n_sweeps == 0) return PIMC_OK;
    // The tuning rule turns the acceptance rate of the last N_skip PROPOSED moves into a step size; a sweep
    // that proposes only one class would shrink the other class's step sizes with no proposals behind it.
    if (h->site_widths && h->tune && !(do_states && do_params))
        return fail(h, PIMC_ESTATE, "step-size tuning needs full sweeps: pimc_sweep_states_only / _params_only are refused while it is on");
    if (((h->t + (unsigned long long)n_sweeps) >> 48) != 0) return fail(h, PIMC_EINVAL, "sweep index exceeds 48 bits");
    OpArgs o{}; o.op = OP_SWEEP; o.h = h; o.n_sweeps = n_sweeps; o.seed = seed; o.do_states = do_states; o.do_params = do_params;
    return dispatch_op(h->model, h->D, h->dtype, o);
}

int recentre(pimc_handle* h) {
    const size_t nx = (size_t)h->C * (h->M + 1) * h->D, np = (size_t)h->C * h->Np;
    const int threads = 256;
    const int bx = (int)std::min<size_t>((nx + threads - 1) / threads, (size_t)h->sm_count * 8), bp = (int)((np + threads - 1) / threads);
    if (h->dtype == 64) {
        widen_kernel<double><<<bx, threads, 0, h->stream>>>((const double*)h->lay.x, h->lay.cx, nx);
        if (np) widen_kernel<double><<<bp, threads, 0, h->stream>>>((const double*)h->lay.p, h->lay.cp, np);
    } else {
        widen_kernel<float><<<bx, threads, 0, h->stream>>>((const float*)h->lay.x, h->lay.cx, nx);
        if (np) widen_kernel<float><<<bp, threads, 0, h->stream>>>((const float*)h->lay.p, h->lay.cp, np);
    }
    h->launches += np ? 2 : 1;
    PIMC_CUDA(h, cudaGetLastError());
    return PIMC_OK;
}

bool finite_all(const double* v, int n) {
    for (int i = 0; i < n; ++i) if (!std::isfinite(v[i])) return false;
    return true;
}

}  // namespace

// ---- latency probes (pimc_latency_selftest): what one inter-CTA message through L2 is made of -------------------------------
namespace {
constexpr int kLatMaxLines = 256, kLatLineStrideWords = 512, kLatReps = 64;      // lines 4 KB apart
// what = 0: every SM (one thread) times a dependent chain of ld.relaxed.gpu on each of n_lines lines: the cost of an L2 HIT from that SM
__global__ void lat_l2map_kernel(unsigned long long* lines, int n_lines, float* out) {
    if (threadIdx.x != 0) return;
    for (int l = 0; l < n_lines; ++l) {
        unsigned long long* p = lines + (size_t)l * kLatLineStrideWords;
        unsigned long long v = 0;
        asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
        const long long t0 = clock64();
        for (int r = 0; r < kLatReps; ++r)
            asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p + (v & 1ull)) : "memory");     // v == 0: same address, dependent
        out[(size_t)blockIdx.x * n_lines + l] = (float)(clock64() - t0) / kLatReps + (float)(v & 1ull);
    }
}
__device__ __forceinline__ void lat_publish(int how, unsigned long long* p, unsigned long long tag) {
    unsigned long long o;
    if (how == 1) asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(tag), "l"(tag) : "memory");
    else if (how == 2) { asm volatile("atom.relaxed.gpu.global.exch.b64 %0, [%1], %2;" : "=l"(o) : "l"(p), "l"(tag) : "memory");
                         asm volatile("atom.relaxed.gpu.global.exch.b64 %0, [%1], %2;" : "=l"(o) : "l"(p + 1), "l"(tag) : "memory"); }
    else if (how == 3) { asm volatile("red.relaxed.gpu.global.max.u64 [%0], %1;" ::"l"(p), "l"(tag) : "memory");
                         asm volatile("red.relaxed.gpu.global.max.u64 [%0], %1;" ::"l"(p + 1), "l"(tag) : "memory"); }
    else if (how == 4) asm volatile("st.volatile.global.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(tag), "l"(tag) : "memory");
    else asm volatile("st.release.gpu.global.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(tag), "l"(tag) : "memory");
}
// what = 1..5: CTA 0 and CTA `peer` play ping-pong with a tagged 16-byte packet (one reader per line: no contention); one-way ticks
__global__ void lat_pingpong_kernel(int how, int first_cta, int peer, int rounds, unsigned long long* box, long long* out) {
    if (threadIdx.x != 0 || ((int)blockIdx.x != first_cta && (int)blockIdx.x != peer)) return;
    const bool first = (int)blockIdx.x == first_cta;
    unsigned long long* mine = box + (first ? 0 : 64);             // the pair's two lines are 512 B apart
    const unsigned long long* theirs = box + (first ? 64 : 0);
    long long t0 = 0;
    for (int r = 1; r <= rounds; ++r) {
        if (r == 11 && first) t0 = clock64();
        if (first) lat_publish(how, mine, (unsigned long long)r);
        unsigned long long a, b, spins = 0;
        do {
            asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "l"(theirs) : "memory");
        } while ((a < (unsigned long long)r || b < (unsigned long long)r) && ++spins < kSpinLimit);
        if (!first) lat_publish(how, mine, (unsigned long long)r);
    }
    if (first) out[0] = (clock64() - t0) / (2 * (rounds - 10));
}
}  // namespace

// ---- device scratch of the no-allocation entry point (pimc_run_host_static) -------------------------------------------------
// A file-scope device array: every GPU that loads libpimc.so holds these 32 MiB until the process exits.  In HOST code the
// name g_static_scratch is only a stand-in for the symbol, NOT a device address (a kernel handed it would fault, or use the
// wrong memory where the GPU can reach host memory): the address on a device comes from cudaGetSymbolAddress with that device
// current, looked up once per device below.  Zero-initialised at load, after that it keeps the last call's contents.
constexpr size_t kStaticScratchBytes = (size_t)32 << 20;
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

namespace {
constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mutex;
void* g_static_addr[kStaticMaxDevices];       // device address of g_static_scratch on device d; nullptr = not looked up yet

int static_scratch_address(void** out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(nullptr, PIMC_ECUDA, "cudaGetDevice: %s (libpimc has no CPU fallback)", cudaGetErrorString(e));
    if (dev < 0 || dev >= kStaticMaxDevices) return fail(nullptr, PIMC_EUNSUPPORTED, "device ordinal %d beyond the %d this entry point keeps addresses for", dev, kStaticMaxDevices);
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[dev]) {
        void* ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_static_scratch);      // device `dev` is current
        if (e != cudaSuccess || !ptr) return fail(nullptr, PIMC_ECUDA, "cudaGetSymbolAddress(g_static_scratch) on device %d: %s", dev, cudaGetErrorString(e));
        if (((uintptr_t)ptr & 255) != 0) return fail(nullptr, PIMC_ECUDA, "static scratch is not 256-byte aligned on device %d", dev);
        g_static_addr[dev] = ptr;
    }
    *out = g_static_addr[dev];
    return PIMC_OK;
}
}  // namespace

extern "C" {

int pimc_model_np(int model, int D) {
    if (model == PIMC_MODEL_HH || model == PIMC_MODEL_HH_CLASSIC) return D == 4 ? 7 : -1;
    if (model == PIMC_MODEL_LINEAR) return (D >= 1 && D <= 4) ? D * D : -1;
    return -1;
}

size_t pimc_workspace_bytes(int model, int D, int L, int M, int n_chains, int dtype) {
    int why;
    if (!shape_ok(model, D, L, M, n_chains, dtype, &why)) return 0;
    return carve(nullptr, D, L, M, pimc_model_np(model, D), n_chains, dtype).bytes;
}

int pimc_init(pimc_handle** out, int model, int D, int L, int M, double dt, double Rm, const double* Rf, const double* p0,
              int n_chains, int dtype, void* workspace, size_t workspace_bytes, void* stream) {
    if (!out) return fail(nullptr, PIMC_EINVAL, "null handle pointer");
    *out = nullptr;
    int why;
    if (!shape_ok(model, D, L, M, n_chains, dtype, &why)) return fail(nullptr, why, "bad or unsupported shape (model=%d D=%d L=%d M=%d chains=%d dtype=%d)", model, D, L, M, n_chains, dtype);
    if (!Rf || !p0) return fail(nullptr, PIMC_EINVAL, "Rf and p0 are required");
    if (!std::isfinite(dt) || !std::isfinite(Rm) || Rm < 0 || !finite_all(Rf, D)) return fail(nullptr, PIMC_EINVAL, "dt, Rm, Rf must be finite (Rm, Rf >= 0)");
    for (int c = 0; c < D; ++c) if (Rf[c] < 0) return fail(nullptr, PIMC_EINVAL, "Rf must be >= 0");
    const int Np = pimc_model_np(model, D);
    if (!finite_all(p0, n_chains * Np)) return fail(nullptr, PIMC_EINVAL, "p0 must be finite");
    const size_t need = carve(nullptr, D, L, M, Np, n_chains, dtype).bytes;
    if (!workspace || ((uintptr_t)workspace & 255) != 0) return fail(nullptr, PIMC_EINVAL, "workspace must be a 256-byte aligned device pointer");
    if (workspace_bytes < need) return fail(nullptr, PIMC_EINVAL, "workspace too small: %zu < %zu", workspace_bytes, need);

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(nullptr, PIMC_ECUDA, "no CUDA device: libpimc has no CPU fallback");
    pimc_handle* h = new (std::nothrow) pimc_handle();
    if (!h) return fail(nullptr, PIMC_ENOMEM, "out of host memory");
    h->model = model; h->D = D; h->L = L; h->M = M; h->Np = Np; h->C = n_chains; h->dtype = dtype;
    h->dt = dt; h->Rm = Rm;
    for (int c = 0; c < D; ++c) h->Rf[c] = Rf[c];
    for (int c = 0; c < kMaxD; ++c) h->wx[c] = 0.0;
    for (int l = 0; l < kMaxNp; ++l) h->wp[l] = 0.0;
    h->stream = (cudaStream_t)stream;
    h->lay = carve((char*)workspace, D, L, M, Np, n_chains, dtype);
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaMemsetAsync(workspace, 0, need, h->stream);
    // parameters and (infinite) bounds
    std::vector<double> lo((size_t)n_chains * Np, -INFINITY), hi((size_t)n_chains * Np, INFINITY);
    if (e == cudaSuccess && Np) {
        if (dtype == 64) e = cudaMemcpyAsync(h->lay.p, p0, sizeof(double) * n_chains * Np, cudaMemcpyHostToDevice, h->stream);
        else {
            std::vector<float> pf(p0, p0 + (size_t)n_chains * Np);
            e = cudaMemcpyAsync(h->lay.p, pf.data(), sizeof(float) * n_chains * Np, cudaMemcpyHostToDevice, h->stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);   // pf is a temporary
        }
        if (e == cudaSuccess) e = cudaMemcpyAsync(h->lay.lo, lo.data(), sizeof(double) * lo.size(), cudaMemcpyHostToDevice, h->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(h->lay.hi, hi.data(), sizeof(double) * hi.size(), cudaMemcpyHostToDevice, h->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);       // host temporaries go out of scope
    }
    if (e != cudaSuccess) {
        fail(nullptr, PIMC_ECUDA, "pimc_init: %s", cudaGetErrorString(e));
        delete h;
        return PIMC_ECUDA;
    }
    *out = h;
    return PIMC_OK;
}

int pimc_set_data(pimc_handle* h, const void* y, const void* I) {
    if (!h) return PIMC_EINVAL;
    if (h->L > 0 && !y) return fail(h, PIMC_EINVAL, "y is required when L > 0");
    if (!aligned32(y) || !aligned32(I)) return fail(h, PIMC_EINVAL, "y and I must be 32-byte aligned device pointers");
    const size_t es = h->dtype == 64 ? 8 : 4;
    if (h->L > 0) PIMC_CUDA(h, cudaMemcpyAsync(h->lay.y, y, (size_t)h->C * (h->M + 1) * h->L * es, cudaMemcpyDeviceToDevice, h->stream));
    if (h->model != PIMC_MODEL_LINEAR && !I) return fail(h, PIMC_EINVAL, "the HH model needs the injected current I");
    h->have_I = I != nullptr;
    if (I) PIMC_CUDA(h, cudaMemcpyAsync(h->lay.I, I, (size_t)h->C * (h->M + 1) * es, cudaMemcpyDeviceToDevice, h->stream));
    h->have_data = true;
    if (h->have_path) return rebuild(h);
    return PIMC_OK;
}

int pimc_set_path(pimc_handle* h, const void* x) {
    if (!h || !x) return fail(h, PIMC_EINVAL, "null argument");
    if (!aligned32(x)) return fail(h, PIMC_EINVAL, "x must be a 32-byte aligned device pointer");
    if (!h->have_data) return fail(h, PIMC_ESTATE, "pimc_set_path before pimc_set_data");
    const size_t es = h->dtype == 64 ? 8 : 4;
    PIMC_CUDA(h, cudaMemcpyAsync(h->lay.x, x, (size_t)h->C * (h->M + 1) * h->D * es, cudaMemcpyDeviceToDevice, h->stream));
    h->have_path = true;
    return rebuild(h);
}

int pimc_set_params(pimc_handle* h, const void* p) {
    if (!h || !p) return fail(h, PIMC_EINVAL, "null argument");
    if (!aligned32(p)) return fail(h, PIMC_EINVAL, "p must be a 32-byte aligned device pointer");
    const size_t es = h->dtype == 64 ? 8 : 4;
    PIMC_CUDA(h, cudaMemcpyAsync(h->lay.p, p, (size_t)h->C * h->Np * es, cudaMemcpyDeviceToDevice, h->stream));
    if (h->have_path) return rebuild(h);
    return PIMC_OK;
}

int pimc_get_path(pimc_handle* h, void* x_out, void* p_out) {
    if (!h) return PIMC_EINVAL;
    if (!aligned32(x_out) || !aligned32(p_out)) return fail(h, PIMC_EINVAL, "x_out and p_out must be 32-byte aligned device pointers");
    const size_t es = h->dtype == 64 ? 8 : 4;
    if (x_out) PIMC_CUDA(h, cudaMemcpyAsync(x_out, h->lay.x, (size_t)h->C * (h->M + 1) * h->D * es, cudaMemcpyDeviceToDevice, h->stream));
    if (p_out) PIMC_CUDA(h, cudaMemcpyAsync(p_out, h->lay.p, (size_t)h->C * h->Np * es, cudaMemcpyDeviceToDevice, h->stream));
    return PIMC_OK;
}

int pimc_get_cache(pimc_handle* h, void* g_out) {
    if (!h || !g_out) return fail(h, PIMC_EINVAL, "null argument");
    if (!h->have_path) return fail(h, PIMC_ESTATE, "no path set");
    const size_t es = h->dtype == 64 ? 8 : 4;
    // the selector lives on the device; chains may differ, so copy chain by chain after reading it back
    std::vector<int> cur(h->C);
    PIMC_CUDA(h, cudaMemcpyAsync(cur.data(), h->lay.cur, sizeof(int) * h->C, cudaMemcpyDeviceToHost, h->stream));
    PIMC_CUDA(h, cudaStreamSynchronize(h->stream));
    const size_t per = (size_t)(h->disc == PIMC_DISC_TRAPEZOID ? h->M + 1 : h->M) * h->D * es;
    for (int c = 0; c < h->C; ++c) {
        const char* src = (const char*)(cur[c] ? h->lay.g1 : h->lay.g0) + per * c;
        PIMC_CUDA(h, cudaMemcpyAsync((char*)g_out + per * c, src, per, cudaMemcpyDeviceToDevice, h->stream));
    }
    return PIMC_OK;
}

int pimc_set_tuning(pimc_handle* h, int enabled, long long n_skip, double f_acc, double alpha) {
    if (!h) return PIMC_EINVAL;
    if (!h->have_prop) return fail(h, PIMC_ESTATE, "pimc_set_tuning before pimc_set_proposal");
    if (!enabled) { h->tune = 0; return PIMC_OK; }                  // step sizes stay as they are
    if (n_skip < 1 || !(f_acc > 0.0 && f_acc < 1.0) || !(alpha >= 0.0 && alpha < 1.0))
        return fail(h, PIMC_EINVAL, "tuning needs n_skip >= 1, 0 < f_acc < 1, 0 <= alpha < 1");
    const size_t nx = (size_t)h->C * (h->M + 1) * h->D, np = (size_t)h->C * h->Np;
    if (!h->site_widths) {                                           // first time: every site starts from the uniform widths
        std::vector<double> w(nx), wp(np);
        for (size_t i = 0; i < nx; ++i) w[i] = h->wx[i % h->D];
        for (size_t i = 0; i < np; ++i) wp[i] = h->wp[i % h->Np];
        PIMC_CUDA(h, cudaMemcpyAsync(h->lay.ws, w.data(), sizeof(double) * nx, cudaMemcpyHostToDevice, h->stream));
        if (np) PIMC_CUDA(h, cudaMemcpyAsync(h->lay.wpd, wp.data(), sizeof(double) * np, cudaMemcpyHostToDevice, h->stream));
        PIMC_CUDA(h, cudaStreamSynchronize(h->stream));
        h->site_widths = true;
    }
    PIMC_CUDA(h, cudaMemsetAsync(h->lay.nacc_s, 0, sizeof(unsigned int) * nx, h->stream));
    if (np) PIMC_CUDA(h, cudaMemsetAsync(h->lay.nacc_p, 0, sizeof(unsigned int) * np, h->stream));
    h->tune = 1; h->tune_skip = (unsigned long long)n_skip; h->f_acc = f_acc; h->alpha = alpha; h->t_tune = h->t;
    return PIMC_OK;
}

int pimc_get_widths(pimc_handle* h, double* ws_out, double* wp_out) {
    if (!h) return PIMC_EINVAL;
    if (!h->have_prop) return fail(h, PIMC_ESTATE, "no proposal widths set");
    const size_t nx = (size_t)h->C * (h->M + 1) * h->D, np = (size_t)h->C * h->Np;
    if (h->site_widths) {
        if (ws_out) PIMC_CUDA(h, cudaMemcpyAsync(ws_out, h->lay.ws, sizeof(double) * nx, cudaMemcpyDeviceToDevice, h->stream));
        if (wp_out && np) PIMC_CUDA(h, cudaMemcpyAsync(wp_out, h->lay.wpd, sizeof(double) * np, cudaMemcpyDeviceToDevice, h->stream));
    } else {
        std::vector<double> w(nx), wp(np);
        for (size_t i = 0; i < nx; ++i) w[i] = h->wx[i % h->D];
        for (size_t i = 0; i < np; ++i) wp[i] = h->wp[i % h->Np];
        if (ws_out) PIMC_CUDA(h, cudaMemcpyAsync(ws_out, w.data(), sizeof(double) * nx, cudaMemcpyHostToDevice, h->stream));
        if (wp_out && np) PIMC_CUDA(h, cudaMemcpyAsync(wp_out, wp.data(), sizeof(double) * np, cudaMemcpyHostToDevice, h->stream));
        PIMC_CUDA(h, cudaStreamSynchronize(h->stream));
    }
    return PIMC_OK;
}

int pimc_set_annealing(pimc_handle* h, double beta0, long long n_cool) {
    if (!h) return PIMC_EINVAL;
    if (!(beta0 > 0.0 && beta0 <= 1.0) || n_cool < 0) return fail(h, PIMC_EINVAL, "annealing needs 0 < beta0 <= 1 and n_cool >= 0");
    h->beta0 = beta0; h->n_cool = (unsigned long long)n_cool; h->t_anneal = h->t;
    return PIMC_OK;
}

int pimc_set_update_mode(pimc_handle* h, int mode) {
    if (!h) return PIMC_EINVAL;
    if (!(mode == PIMC_UPDATE_JOINT || mode == PIMC_UPDATE_COMPONENTWISE)) return fail(h, PIMC_EINVAL, "unknown update mode %d", mode);
    h->update_mode = mode;
    return PIMC_OK;
}

int pimc_set_discretisation(pimc_handle* h, int disc) {
    if (!h) return PIMC_EINVAL;
    if (!(disc == PIMC_DISC_RK4MAP || disc == PIMC_DISC_TRAPEZOID)) return fail(h, PIMC_EINVAL, "unknown discretisation %d", disc);
    h->disc = disc;
    if (h->have_path) return rebuild(h);
    return PIMC_OK;
}

int pimc_set_proposal(pimc_handle* h, const double* w_state, const double* w_param, int kind) {
    if (!h || !w_state) return fail(h, PIMC_EINVAL, "null argument");
    if (!(kind == PIMC_PROPOSAL_GAUSSIAN || kind == PIMC_PROPOSAL_UNIFORM)) return fail(h, PIMC_EINVAL, "unknown proposal kind");
    for (int c = 0; c < h->D; ++c) if (!(w_state[c] >= 0) || !std::isfinite(w_state[c])) return fail(h, PIMC_EINVAL, "w_state must be finite and >= 0");
    if (w_param) for (int l = 0; l < h->Np; ++l) if (!(w_param[l] >= 0) || !std::isfinite(w_param[l])) return fail(h, PIMC_EINVAL, "w_param must be finite and >= 0");
    for (int c = 0; c < h->D; ++c) h->wx[c] = w_state[c];
    for (int l = 0; l < h->Np; ++l) h->wp[l] = w_param ? w_param[l] : 0.0;
    h->kind = kind;
    h->have_prop = true;
    h->site_widths = false; h->tune = 0;      // uniform step sizes again
    return PIMC_OK;
}

int pimc_set_bounds(pimc_handle* h, const double* lo, const double* hi) {
    if (!h || !lo || !hi) return fail(h, PIMC_EINVAL, "null argument");
    const size_t n = (size_t)h->C * h->Np;
    for (size_t i = 0; i < n; ++i) if (!(lo[i] <= hi[i])) return fail(h, PIMC_EINVAL, "bounds need lo <= hi");
    PIMC_CUDA(h, cudaMemcpyAsync(h->lay.lo, lo, sizeof(double) * n, cudaMemcpyHostToDevice, h->stream));
    PIMC_CUDA(h, cudaMemcpyAsync(h->lay.hi, hi, sizeof(double) * n, cudaMemcpyHostToDevice, h->stream));
    PIMC_CUDA(h, cudaStreamSynchronize(h->stream));   // lo/hi are pageable host memory owned by the caller
    return PIMC_OK;
}

int pimc_set_accum(pimc_handle* h, int enabled, long long n_skip) {
    if (!h) return PIMC_EINVAL;
    if (n_skip < 1) return fail(h, PIMC_EINVAL, "n_skip must be >= 1");
    if (enabled && !h->accum) h->t_enable = h->t;
    h->accum = enabled ? 1 : 0;
    h->n_skip = (unsigned long long)n_skip;
    return PIMC_OK;
}

int pimc_reset_moments(pimc_handle* h) {
    if (!h) return PIMC_EINVAL;
    if (!h->have_path) return fail(h, PIMC_ESTATE, "no path set");
    const size_t nx = (size_t)h->C * (h->M + 1) * h->D, np = (size_t)h->C * h->Np;
    PIMC_CUDA(h, cudaMemsetAsync(h->lay.S1x, 0, sizeof(double) * nx, h->stream));
    PIMC_CUDA(h, cudaMemsetAsync(h->lay.S2x, 0, sizeof(double) * nx, h->stream));
    if (np) {
        PIMC_CUDA(h, cudaMemsetAsync(h->lay.S1p, 0, sizeof(double) * np, h->stream));
        PIMC_CUDA(h, cudaMemsetAsync(h->lay.S2p, 0, sizeof(double) * np, h->stream));
    }
    if (h->n_sel) PIMC_CUDA(h, cudaMemsetAsync(h->lay.hist, 0, sizeof(unsigned long long) * (size_t)h->C * h->n_sel * (h->nbins + 2), h->stream));
    if (h->resid_acc) PIMC_CUDA(h, cudaMemsetAsync(h->resid_acc, 0, sizeof(double) * (size_t)h->C * (2 * (size_t)h->M * h->D + 2 * (size_t)(h->M + 1) * h->L), h->stream));
    h->n_samples = 0;
    h->t_enable = h->t;
    return recentre(h);
}

int pimc_sweep(pimc_handle* h, long long n_sweeps, unsigned long long seed) { return sweep_common(h, n_sweeps, seed, 1, 1); }
int pimc_sweep_states_only(pimc_handle* h, long long n_sweeps, unsigned long long seed) { return sweep_common(h, n_sweeps, seed, 1, 0); }
int pimc_sweep_params_only(pimc_handle* h, long long n_sweeps, unsigned long long seed) { return sweep_common(h, n_sweeps, seed, 0, 1); }

int pimc_moments(pimc_handle* h, double* out, unsigned long long* n_samples_host) {
    if (!h || !out) return fail(h, PIMC_EINVAL, "null argument");
    if (!aligned32(out)) return fail(h, PIMC_EINVAL, "out must be a 32-byte aligned device pointer");
    const size_t nx = (size_t)(h->M + 1) * h->D;
    const size_t total = (size_t)h->C * (nx + h->Np);
    const int threads = 256;
    const int blocks = (int)std::min<size_t>((total + threads - 1) / threads, (size_t)h->sm_count * 8);
    moments_kernel<<<blocks, threads, 0, h->stream>>>(h->lay.cx, h->lay.S1x, h->lay.S2x, h->lay.cp, h->lay.S1p, h->lay.S2p, nx, h->Np,
                                                      h->C, (double)h->n_samples, out);
    h->launches++;
    PIMC_CUDA(h, cudaGetLastError());
    if (n_samples_host) *n_samples_host = h->n_samples;
    return PIMC_OK;
}

int pimc_stats(pimc_handle* h, unsigned long long* acc_out) {
    if (!h || !acc_out) return fail(h, PIMC_EINVAL, "null argument");
    PIMC_CUDA(h, cudaMemcpyAsync(acc_out, h->lay.counters, sizeof(unsigned long long) * (size_t)h->C * 2 * (h->D + h->Np),
                                 cudaMemcpyDeviceToDevice, h->stream));
    return PIMC_OK;
}

int pimc_hist_config(pimc_handle* h, int n_sel, const int* site, const int* comp, const double* lo, const double* hi, int nbins) {
    if (!h) return PIMC_EINVAL;
    if (n_sel < 0 || n_sel > kMaxHistSel) return fail(h, PIMC_EINVAL, "n_sel must be in [0,%d]", kMaxHistSel);
    if (n_sel == 0) { h->n_sel = 0; return PIMC_OK; }
    if (!site || !comp || !lo || !hi || nbins < 1) return fail(h, PIMC_EINVAL, "bad histogram arguments");
    if ((size_t)h->C * n_sel * (nbins + 2) > kMaxHistWords) return fail(h, PIMC_EINVAL, "histogram storage exceeds %zu counters", kMaxHistWords);
    std::vector<double> width(n_sel);
    for (int i = 0; i < n_sel; ++i) {
        if (site[i] > h->M || site[i] < -1) return fail(h, PIMC_EINVAL, "histogram site out of range");
        if (comp[i] < 0 || comp[i] >= (site[i] < 0 ? h->Np : h->D)) return fail(h, PIMC_EINVAL, "histogram component out of range");
        if (!(lo[i] < hi[i])) return fail(h, PIMC_EINVAL, "histogram range needs lo < hi");
        width[i] = (hi[i] - lo[i]) / nbins;
    }
    PIMC_CUDA(h, cudaMemcpyAsync(h->lay.hsite, site, sizeof(int) * n_sel, cudaMemcpyHostToDevice, h->stream));
    PIMC_CUDA(h, cudaMemcpyAsync(h->lay.hcomp, comp, sizeof(int) * n_sel, cudaMemcpyHostToDevice, h->stream));
    PIMC_CUDA(h, cudaMemcpyAsync(h->lay.hlo, lo, sizeof(double) * n_sel, cudaMemcpyHostToDevice, h->stream));
    PIMC_CUDA(h, cudaMemcpyAsync(h->lay.hhi, hi, sizeof(double) * n_sel, cudaMemcpyHostToDevice, h->stream));
    PIMC_CUDA(h, cudaMemcpyAsync(h->lay.hwidth, width.data(), sizeof(double) * n_sel, cudaMemcpyHostToDevice, h->stream));
    PIMC_CUDA(h, cudaMemsetAsync(h->lay.hist, 0, sizeof(unsigned long long) * (size_t)h->C * n_sel * (nbins + 2), h->stream));
    PIMC_CUDA(h, cudaStreamSynchronize(h->stream));
    h->n_sel = n_sel; h->nbins = nbins;
    return PIMC_OK;
}

int pimc_hist(pimc_handle* h, unsigned long long* counts_out) {
    if (!h || !counts_out) return fail(h, PIMC_EINVAL, "null argument");
    if (!h->n_sel) return fail(h, PIMC_ESTATE, "no histogram configured");
    PIMC_CUDA(h, cudaMemcpyAsync(counts_out, h->lay.hist, sizeof(unsigned long long) * (size_t)h->C * h->n_sel * (h->nbins + 2),
                                 cudaMemcpyDeviceToDevice, h->stream));
    return PIMC_OK;
}

int pimc_debug_trace(pimc_handle* h, void* dA_out, unsigned char* acc_out, void* xprop_out, void* dA_param, unsigned char* acc_param,
                     void* pprop_out) {
    if (!h) return PIMC_EINVAL;
    if (!aligned32(dA_out) || !aligned32(xprop_out) || !aligned32(dA_param) || !aligned32(pprop_out))
        return fail(h, PIMC_EINVAL, "trace arrays must be 32-byte aligned device pointers");
    h->tr_dA = dA_out; h->tr_acc = acc_out; h->tr_xprop = xprop_out; h->tr_dAp = dA_param; h->tr_accp = acc_param; h->tr_pprop = pprop_out;
    return PIMC_OK;
}

int pimc_set_launch(pimc_handle* h, int ctas_per_chain, int threads_per_cta) {
    if (!h) return PIMC_EINVAL;
    if (ctas_per_chain < 0 || ctas_per_chain > kMaxCtasPerChain) return fail(h, PIMC_EINVAL, "ctas_per_chain out of range");
    if (threads_per_cta != 0 && (threads_per_cta % 32 != 0 || threads_per_cta < 32 || threads_per_cta > kMaxThreads))
        return fail(h, PIMC_EINVAL, "threads_per_cta must be 0 or a multiple of 32 in [32,%d]", kMaxThreads);
    const int G0 = h->G_user, T0 = h->T_user;
    h->G_user = ctas_per_chain; h->T_user = threads_per_cta;
    LaunchShape ls;
    OpArgs o{}; o.op = OP_SHAPE; o.h = h; o.ls = &ls;
    const int rc = dispatch_op(h->model, h->D, h->dtype, o);
    if (rc != PIMC_OK) { h->G_user = G0; h->T_user = T0; }
    return rc;
}

int pimc_get_launch(pimc_handle* h, int* ctas_per_chain, int* threads_per_cta, int* tile_sites, int* smem_bytes) {
    if (!h) return PIMC_EINVAL;
    LaunchShape ls;
    OpArgs o{}; o.op = OP_SHAPE; o.h = h; o.ls = &ls;
    const int rc = dispatch_op(h->model, h->D, h->dtype, o);
    if (rc != PIMC_OK) return rc;
    if (ctas_per_chain) *ctas_per_chain = ls.G;
    if (threads_per_cta) *threads_per_cta = ls.T;
    if (tile_sites) *tile_sites = ls.tile;
    if (smem_bytes) *smem_bytes = (int)ls.smem;
    return PIMC_OK;
}

int pimc_set_engine(pimc_handle* h, int engine, int halo) {
    if (!h) return PIMC_EINVAL;
    if (engine < PIMC_ENGINE_AUTO || engine > PIMC_ENGINE_TILE_MC) return fail(h, PIMC_EINVAL, "unknown engine");
    if (halo < -1 || halo > kTileHaloMax || (halo > 0 && (halo & 1))) return fail(h, PIMC_EINVAL, "halo must be -1 (automatic) or an even number in [0,%d]", kTileHaloMax);
    const int e0 = h->engine_user, h0 = h->halo_user;
    h->engine_user = engine; h->halo_user = halo;
    LaunchShape ls;
    OpArgs o{}; o.op = OP_SHAPE; o.h = h; o.ls = &ls;
    const int rc = dispatch_op(h->model, h->D, h->dtype, o);
    if (rc != PIMC_OK) { h->engine_user = e0; h->halo_user = h0; }
    return rc;
}

int pimc_get_engine(pimc_handle* h, int* engine, int* halo) {
    if (!h) return PIMC_EINVAL;
    LaunchShape ls;
    OpArgs o{}; o.op = OP_SHAPE; o.h = h; o.ls = &ls;
    const int rc = dispatch_op(h->model, h->D, h->dtype, o);
    if (rc != PIMC_OK) return rc;
    if (engine) *engine = ls.engine;
    if (halo) *halo = ls.h;
    return PIMC_OK;
}

int pimc_param_trace(pimc_handle* h, void* out, long long capacity) {
    if (!h) return PIMC_EINVAL;
    if (out && (capacity < 1 || !aligned32(out))) return fail(h, PIMC_EINVAL, "parameter record needs capacity >= 1 and a 32-byte aligned device pointer");
    if (out && h->Np == 0) return fail(h, PIMC_EUNSUPPORTED, "the model has no parameters");
    h->ptrace = out; h->ptrace_cap = out ? capacity : 0;
    return PIMC_OK;
}

int pimc_residuals(pimc_handle* h, void* eps_out, void* delta_out) {
    if (!h) return PIMC_EINVAL;
    if (!h->have_path) return fail(h, PIMC_ESTATE, "no path set");
    if (!aligned32(eps_out) || !aligned32(delta_out)) return fail(h, PIMC_EINVAL, "outputs must be 32-byte aligned device pointers");
    const size_t total = (size_t)h->C * (h->M + 1);
    const int threads = 256;
    const int blocks = (int)std::min<size_t>((total + threads - 1) / threads, (size_t)h->sm_count * 8);
    const int nc = h->disc == PIMC_DISC_TRAPEZOID ? h->M + 1 : h->M;
    if (h->dtype == 64)
        residual_kernel<double><<<blocks, threads, 0, h->stream>>>((const double*)h->lay.x, (const double*)h->lay.g0, (const double*)h->lay.g1, h->lay.cur,
                                                                   (const double*)h->lay.y, h->M, h->D, h->L, nc, h->disc, h->C, (double*)eps_out, (double*)delta_out, nullptr);
    else
        residual_kernel<float><<<blocks, threads, 0, h->stream>>>((const float*)h->lay.x, (const float*)h->lay.g0, (const float*)h->lay.g1, h->lay.cur,
                                                                  (const float*)h->lay.y, h->M, h->D, h->L, nc, h->disc, h->C, (float*)eps_out, (float*)delta_out, nullptr);
    h->launches++;
    PIMC_CUDA(h, cudaGetLastError());
    return PIMC_OK;
}

int pimc_set_residual_stats(pimc_handle* h, double* acc) {
    if (!h) return PIMC_EINVAL;
    if (!aligned32(acc)) return fail(h, PIMC_EINVAL, "acc must be a 32-byte aligned device pointer");
    h->resid_acc = acc;
    if (acc) PIMC_CUDA(h, cudaMemsetAsync(acc, 0, sizeof(double) * (size_t)h->C * (2 * (size_t)h->M * h->D + 2 * (size_t)(h->M + 1) * h->L), h->stream));
    return PIMC_OK;
}

int pimc_residual_stats(pimc_handle* h, double* out) {
    if (!h || !out) return fail(h, PIMC_EINVAL, "null argument");
    if (!h->resid_acc) return fail(h, PIMC_ESTATE, "residual statistics are not enabled");
    if (!aligned32(out)) return fail(h, PIMC_EINVAL, "out must be a 32-byte aligned device pointer");
    const size_t ne = (size_t)h->M * h->D, nd = (size_t)(h->M + 1) * h->L;
    const size_t total = (size_t)h->C * (ne + nd);
    const int threads = 256;
    const int blocks = (int)std::min<size_t>((total + threads - 1) / threads, (size_t)h->sm_count * 8);
    residual_stats_kernel<<<blocks, threads, 0, h->stream>>>(h->resid_acc, ne, nd, h->C, (double)h->n_samples, out);
    h->launches++;
    PIMC_CUDA(h, cudaGetLastError());
    return PIMC_OK;
}

int pimc_set_exchange(pimc_handle* h, int first_poll_hold_cycles) {
    if (!h) return PIMC_EINVAL;
    if (first_poll_hold_cycles < 0 || first_poll_hold_cycles > 100000) return fail(h, PIMC_EINVAL, "first_poll_hold_cycles must be in [0, 100000]");
    h->ar_hold = first_poll_hold_cycles;
    return PIMC_OK;
}

int pimc_fault(pimc_handle* h, int* fault_host) {
    if (!h || !fault_host) return fail(h, PIMC_EINVAL, "null argument");
    PIMC_CUDA(h, cudaMemcpyAsync(fault_host, h->lay.fault, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    PIMC_CUDA(h, cudaStreamSynchronize(h->stream));
    if (*fault_host) return fail(h, PIMC_ECUDA, "a hand-off between CTAs was never delivered (fault flag %d)", *fault_host);
    return PIMC_OK;
}

unsigned long long pimc_sweep_index(const pimc_handle* h) { return h ? h->t : 0; }
int pimc_set_sweep_index(pimc_handle* h, unsigned long long t) {
    if (!h) return PIMC_EINVAL;
    if ((t >> 48) != 0) return fail(h, PIMC_EINVAL, "sweep index exceeds 48 bits");
    // The accumulation, tuning and annealing schedules count sweeps from the index at which they were switched on: moving the
    // index below one of those origins would wrap the unsigned differences (sample count, adjustment sweeps, beta) silently.
    if (h->accum && t < h->t_enable) return fail(h, PIMC_ESTATE, "sweep index below the sweep at which accumulation was enabled (disable or reset first)");
    if (h->site_widths && h->tune && t < h->t_tune) return fail(h, PIMC_ESTATE, "sweep index below the sweep at which step-size tuning was enabled");
    if (h->n_cool != 0 && t < h->t_anneal) return fail(h, PIMC_ESTATE, "sweep index below the sweep at which annealing was enabled");
    h->t = t;
    return PIMC_OK;
}
unsigned long long pimc_launch_count(const pimc_handle* h) { return h ? h->launches : 0; }

// layout of the device scratch of pimc_run_host: staging copies of x, y, I, p, the moments read-out, then the handle's workspace
namespace {
struct HostRunLayout { size_t o_x, o_y, o_I, o_p, o_m, o_ws, ws, total, nx, ny, nI, nmom; };
HostRunLayout host_run_layout(int model, int D, int L, int M, int n_chains, int dtype) {
    HostRunLayout q{};
    const int Np = pimc_model_np(model, D);
    const size_t es = dtype == 64 ? 8 : 4;
    auto up = [](size_t v) { return (v + 255) & ~(size_t)255; };
    q.nx = (size_t)n_chains * (M + 1) * D; q.ny = (size_t)n_chains * (M + 1) * (L > 0 ? L : 1); q.nI = (size_t)n_chains * (M + 1);
    q.nmom = (size_t)n_chains * (2 * (size_t)(M + 1) * D + 2 * (size_t)Np);
    q.ws = pimc_workspace_bytes(model, D, L, M, n_chains, dtype);
    q.o_x = 0; q.o_y = q.o_x + up(q.nx * es); q.o_I = q.o_y + up(q.ny * es); q.o_p = q.o_I + up(q.nI * es);
    q.o_m = q.o_p + up((size_t)n_chains * Np * es); q.o_ws = q.o_m + up(q.nmom * 8);
    q.total = q.o_ws + q.ws;
    return q;
}
}  // namespace

size_t pimc_run_host_workspace_bytes(int model, int D, int L, int M, int n_chains, int dtype) {
    int why;
    if (!shape_ok(model, D, L, M, n_chains, dtype, &why)) return 0;
    return host_run_layout(model, D, L, M, n_chains, dtype).total;
}

int pimc_run_host(int model, int D, int L, int M, double dt, double Rm, const double* Rf, int n_chains, int dtype, const void* y,
                  const void* I, const void* x0, const void* p0, const double* w_state, const double* w_param, const double* lo,
                  const double* hi, int proposal_kind, long long n_burn, long long n_sweeps, unsigned long long seed, double* moments_out,
                  void* x_out, void* p_out) {
    return pimc_run_host_ws(model, D, L, M, dt, Rm, Rf, n_chains, dtype, y, I, x0, p0, w_state, w_param, lo, hi, proposal_kind, n_burn,
                            n_sweeps, seed, moments_out, x_out, p_out, nullptr, 0);
}

int pimc_run_host_ws(int model, int D, int L, int M, double dt, double Rm, const double* Rf, int n_chains, int dtype, const void* y,
                     const void* I, const void* x0, const void* p0, const double* w_state, const double* w_param, const double* lo,
                     const double* hi, int proposal_kind, long long n_burn, long long n_sweeps, unsigned long long seed, double* moments_out,
                     void* x_out, void* p_out, void* dev_scratch, size_t dev_scratch_bytes) {
    int why;
    if (!shape_ok(model, D, L, M, n_chains, dtype, &why)) return fail(nullptr, why, "bad or unsupported shape");
    if (!x0 || !p0 || !w_state || !moments_out || (L > 0 && !y)) return fail(nullptr, PIMC_EINVAL, "null argument");
    const int Np = pimc_model_np(model, D);
    const size_t es = dtype == 64 ? 8 : 4;
    const HostRunLayout q = host_run_layout(model, D, L, M, n_chains, dtype);
    const size_t nx = q.nx, ny = q.ny, nI = q.nI, nmom = q.nmom, ws = q.ws, o_x = q.o_x, o_y = q.o_y, o_I = q.o_I, o_p = q.o_p, o_m = q.o_m, o_ws = q.o_ws;
    char* dev = nullptr;
    const bool own = dev_scratch == nullptr;
    if (own) {
        if (cudaMalloc(&dev, q.total) != cudaSuccess) return fail(nullptr, PIMC_ENOMEM, "cudaMalloc of %zu bytes failed", q.total);
    } else {
        if (((uintptr_t)dev_scratch & 255) != 0 || dev_scratch_bytes < q.total)
            return fail(nullptr, PIMC_EINVAL, "device scratch must be 256-byte aligned and at least %zu bytes", q.total);
        dev = (char*)dev_scratch;
    }
    pimc_handle* h = nullptr;
    int rc = PIMC_OK;
    cudaError_t e = cudaSuccess;
    // parameters as doubles for pimc_init (host side)
    std::vector<double> p0d((size_t)n_chains * Np);
    for (size_t i = 0; i < p0d.size(); ++i) p0d[i] = dtype == 64 ? ((const double*)p0)[i] : (double)((const float*)p0)[i];
    do {
        if ((e = cudaMemcpyAsync(dev + o_x, x0, nx * es, cudaMemcpyHostToDevice, 0)) != cudaSuccess) break;
        if (L > 0 && (e = cudaMemcpyAsync(dev + o_y, y, ny * es, cudaMemcpyHostToDevice, 0)) != cudaSuccess) break;
        if (I && (e = cudaMemcpyAsync(dev + o_I, I, nI * es, cudaMemcpyHostToDevice, 0)) != cudaSuccess) break;
        if ((rc = pimc_init(&h, model, D, L, M, dt, Rm, Rf, p0d.data(), n_chains, dtype, dev + o_ws, ws, nullptr)) != PIMC_OK) break;
        if ((rc = pimc_set_data(h, dev + o_y, I ? dev + o_I : nullptr)) != PIMC_OK) break;
        if ((rc = pimc_set_proposal(h, w_state, w_param, proposal_kind)) != PIMC_OK) break;
        if (lo && hi && (rc = pimc_set_bounds(h, lo, hi)) != PIMC_OK) break;
        if ((rc = pimc_set_path(h, dev + o_x)) != PIMC_OK) break;
        if ((rc = pimc_sweep(h, n_burn, seed)) != PIMC_OK) break;
        if ((rc = pimc_set_accum(h, 1, 1)) != PIMC_OK) break;
        if ((rc = pimc_reset_moments(h)) != PIMC_OK) break;
        if ((rc = pimc_sweep(h, n_sweeps, seed)) != PIMC_OK) break;
        if ((rc = pimc_moments(h, (double*)(dev + o_m), nullptr)) != PIMC_OK) break;
        if ((e = cudaMemcpyAsync(moments_out, dev + o_m, nmom * 8, cudaMemcpyDeviceToHost, 0)) != cudaSuccess) break;
        if (x_out || p_out) {
            if ((rc = pimc_get_path(h, x_out ? dev + o_x : nullptr, p_out ? dev + o_p : nullptr)) != PIMC_OK) break;
            if (x_out && (e = cudaMemcpyAsync(x_out, dev + o_x, nx * es, cudaMemcpyDeviceToHost, 0)) != cudaSuccess) break;
            if (p_out && (e = cudaMemcpyAsync(p_out, dev + o_p, (size_t)n_chains * Np * es, cudaMemcpyDeviceToHost, 0)) != cudaSuccess) break;
        }
        if (rc == PIMC_OK) {                       // a lost hand-off must not pass for a result
            int flt = 0;
            if ((rc = pimc_fault(h, &flt)) != PIMC_OK) break;
        }
        e = cudaStreamSynchronize(0);
    } while (0);
    if (rc != PIMC_OK && h) g_static_error = h->err;
    if (e != cudaSuccess) { rc = fail(nullptr, PIMC_ECUDA, "pimc_run_host: %s", cudaGetErrorString(e)); }
    if (h) pimc_destroy(h);
    if (own) cudaFree(dev);
    return rc;
}

size_t pimc_static_scratch_bytes(void) { return kStaticScratchBytes; }

// pimc_run_host with ALL device memory taken from the static array above: no cudaMalloc, no cudaFree, no allocating library
// routine anywhere on the path (pimc_run_host_ws with a caller buffer never allocates device memory; pimc_init clears the
// workspace it carves -- epochs, mailbox tags, counters, moment sums must start at zero -- with a cudaMemsetAsync on the stream).
int pimc_run_host_static(int model, int D, int L, int M, double dt, double Rm, const double* Rf, int n_chains, int dtype, const void* y,
                         const void* I, const void* x0, const void* p0, const double* w_state, const double* w_param, const double* lo,
                         const double* hi, int proposal_kind, long long n_burn, long long n_sweeps, unsigned long long seed,
                         double* moments_out, void* x_out, void* p_out) {
    int why;
    if (!shape_ok(model, D, L, M, n_chains, dtype, &why)) return fail(nullptr, why, "bad or unsupported shape");
    const size_t need = host_run_layout(model, D, L, M, n_chains, dtype).total;
    if (need > kStaticScratchBytes)
        return fail(nullptr, PIMC_EUNSUPPORTED, "pimc_run_host_static: this shape needs %zu bytes of device scratch, the static array holds %zu "
                    "(pimc_static_scratch_bytes); use pimc_run_host_ws with a buffer of your own", need, kStaticScratchBytes);
    void* scratch = nullptr;
    const int rc = static_scratch_address(&scratch);
    if (rc != PIMC_OK) return rc;
    return pimc_run_host_ws(model, D, L, M, dt, Rm, Rf, n_chains, dtype, y, I, x0, p0, w_state, w_param, lo, hi, proposal_kind, n_burn,
                            n_sweeps, seed, moments_out, x_out, p_out, scratch, kStaticScratchBytes);
}

int pimc_rng_selftest(const unsigned int* ctrs, unsigned long long n, unsigned int key0, unsigned int key1, unsigned int* out,
                      double* u_prop, double* u_acc, double* z, void* stream) {
    if (!ctrs) return fail(nullptr, PIMC_EINVAL, "null argument");
    if (n == 0) return PIMC_OK;
    const int threads = 256;
    const int blocks = (int)std::min<unsigned long long>((n + threads - 1) / threads, (unsigned long long)sm_count_now() * 8);
    rng_selftest_kernel<<<blocks, threads, 0, (cudaStream_t)stream>>>(ctrs, n, key0, key1, out, u_prop, u_acc, z);
    PIMC_CUDA(nullptr, cudaGetLastError());
    return PIMC_OK;
}

int pimc_step_selftest(int model, int D, int dtype, const void* x, const void* p, const void* I0, const void* I1, double dt,
                       unsigned long long n, void* g_out, void* stream) {
    if (!x || !p || !g_out) return fail(nullptr, PIMC_EINVAL, "null argument");
    if (pimc_model_np(model, D) < 0 || !(dtype == 64 || dtype == 32)) return fail(nullptr, PIMC_EUNSUPPORTED, "unsupported model / D / dtype");
    if (n == 0) return PIMC_OK;
    OpArgs o{}; o.op = OP_STEP; o.h = nullptr; o.x = x; o.p = p; o.I0 = I0; o.I1 = I1; o.dt = dt; o.n = n; o.g = g_out; o.stream = stream;
    return dispatch_op(model, D, dtype, o);
}

int pimc_math_selftest(const double* x, unsigned long long n, double* out, void* stream) {
    if (!x || !out) return fail(nullptr, PIMC_EINVAL, "null argument");
    if (n == 0) return PIMC_OK;
    const int threads = 256;
    const int blocks = (int)std::min<unsigned long long>((n + threads - 1) / threads, (unsigned long long)sm_count_now() * 8);
    math_selftest_kernel<<<blocks, threads, 0, (cudaStream_t)stream>>>(x, n, out);
    PIMC_CUDA(nullptr, cudaGetLastError());
    return PIMC_OK;
}

int pimc_fp64_peak_selftest(int millis, double* lane_fma_per_s) {
    if (!lane_fma_per_s || millis < 1) return fail(nullptr, PIMC_EINVAL, "bad argument");
    int dev = 0, sms = 0;
    PIMC_CUDA(nullptr, cudaGetDevice(&dev));
    PIMC_CUDA(nullptr, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double* sink = nullptr;
    PIMC_CUDA(nullptr, cudaMalloc(&sink, 64));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int threads = 1024, iters = 40000;
    fp64_peak_kernel<<<sms, threads>>>(sink, iters, 1.0000001, 1e-9);   // warm-up
    cudaDeviceSynchronize();
    double best = 0.0, elapsed = 0.0;
    while (elapsed < (double)millis) {
        cudaEventRecord(e0);
        fp64_peak_kernel<<<sms, threads>>>(sink, iters, 1.0000001, 1e-9);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        elapsed += ms;
        const double rate = (double)sms * threads * 8.0 * iters / (ms * 1e-3);
        if (rate > best) best = rate;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink);
    PIMC_CUDA(nullptr, cudaGetLastError());
    *lane_fma_per_s = best;
    return PIMC_OK;
}

int pimc_exchange_selftest(int mode, int n_ctas, int threads, int rounds, int work, double* cycles_per_round_host,
                           double* max_abs_err_host, int* n_distinct_host) {
    if (!cycles_per_round_host || !max_abs_err_host || !n_distinct_host) return fail(nullptr, PIMC_EINVAL, "null argument");
    if (mode < -1 || (mode > 10 && mode < 100) || mode > 140 || threads < 32 || threads > 256 || threads % 32 != 0 || rounds < 2 || work < 0)
        return fail(nullptr, PIMC_EINVAL, "bad argument");
    int dev = 0, sms = 0;
    PIMC_CUDA(nullptr, cudaGetDevice(&dev));
    PIMC_CUDA(nullptr, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (n_ctas == 0) n_ctas = sms;
    if (n_ctas < 1 || n_ctas > sms || n_ctas > kXchgMaxCtas) return fail(nullptr, PIMC_EINVAL, "n_ctas must be in [1, SM count]");
    const size_t smem = 100 * 1024;               // one CTA per SM, as in the sweep launches
    PIMC_CUDA(nullptr, cudaFuncSetAttribute((const void*)xchg_selftest_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const size_t n_ar = (size_t)2 * kTileMaxCtas * kArSlotWords;
    const size_t n_inbox = (size_t)2 * kTileMaxCtas * kTileMaxCtas * 2;
    const size_t bytes = (kXchgWords + n_ar) * 8 + 256 + (size_t)n_ctas * 8 + 128 + 256 + n_inbox * 8;
    char* devp = nullptr;
    PIMC_CUDA(nullptr, cudaMalloc(&devp, bytes));
    cudaMemset(devp, 0, bytes);
    unsigned long long* mbox = (unsigned long long*)devp;
    unsigned long long* ar = mbox + kXchgWords;
    int* fault = (int*)(ar + n_ar);
    double* out_tot = (double*)((char*)fault + 256);
    long long* out_cycles = (long long*)(out_tot + n_ctas);
    double* sink = (double*)(out_cycles + 6);
    unsigned long long* inbox = (unsigned long long*)(((uintptr_t)(sink + 2) + 255) & ~(uintptr_t)255);
    const int warm = rounds / 4;
    void* params[] = {&mode, &rounds, (void*)&warm, &work, &mbox, &ar, &fault, &out_tot, &out_cycles, &sink, &inbox};
    cudaError_t e = cudaLaunchCooperativeKernel((const void*)xchg_selftest_kernel, dim3((unsigned)n_ctas), dim3((unsigned)threads), params, smem, 0);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    std::vector<double> tot(n_ctas);
    long long cyc = 0;
    int flt = 0;
    if (e == cudaSuccess) e = cudaMemcpy(tot.data(), out_tot, sizeof(double) * n_ctas, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(&cyc, out_cycles, sizeof cyc, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess && (mode == 0 || mode == 6) && getenv("PIMC_XCHG_PHASES")) {
        long long ph[4];
        cudaMemcpy(ph, out_cycles, sizeof ph, cudaMemcpyDeviceToHost);
        const double d = (double)n_ctas * (rounds - warm);
        fprintf(stderr, "phases (mean over CTAs): block sum 1 %.0f, store+poll %.0f, block sum 2 %.0f cycles\n", ph[1] / d, ph[2] / d, ph[3] / d);
    }
    if (e == cudaSuccess) e = cudaMemcpy(&flt, fault, sizeof flt, cudaMemcpyDeviceToHost);
    cudaFree(devp);
    if (e != cudaSuccess) return fail(nullptr, PIMC_ECUDA, "pimc_exchange_selftest: %s", cudaGetErrorString(e));
    if (flt) return fail(nullptr, PIMC_ECUDA, "pimc_exchange_selftest: a packet was never delivered");
    *cycles_per_round_host = (double)cyc / (double)(rounds - warm);
    // expected total of the last round (modes 0-2), in long double on the host
    long double expect = 0.0L;
    for (int b = 0; b < n_ctas; ++b)
        for (int t = 0; t < threads; ++t) expect += (long double)((double)((b * 131 + t * 7 + (rounds - 1) * 13) % 1000 - 500) * 0.001);
    double worst = 0.0;
    int distinct = 1;
    for (int b = 0; b < n_ctas; ++b) {
        if (mode >= 0 && mode != 3 && (mode < 7 || mode >= 10)) worst = std::max(worst, (double)fabsl((long double)tot[b] - expect));
        if (b > 0 && std::memcmp(&tot[b], &tot[0], sizeof(double)) != 0) distinct++;
    }
    *max_abs_err_host = worst;
    *n_distinct_host = (mode >= 0 && mode != 3 && (mode < 7 || mode >= 10)) ? distinct : 1;
    return PIMC_OK;
}

int pimc_latency_selftest(int what, int arg, double* out_host, int n_out) {
    if (!out_host || n_out < 5 || what < 0 || what > 6) return fail(nullptr, PIMC_EINVAL, "bad argument");
    int dev = 0, sms = 0;
    PIMC_CUDA(nullptr, cudaGetDevice(&dev));
    PIMC_CUDA(nullptr, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    for (int k = 0; k < n_out; ++k) out_host[k] = 0.0;
    const size_t smem = 100 * 1024;               // one CTA per SM
    if (what == 0) {
        const int n_lines = arg <= 0 ? 128 : arg;
        if (n_lines > kLatMaxLines) return fail(nullptr, PIMC_EINVAL, "at most %d lines", kLatMaxLines);
        unsigned long long* lines = nullptr;
        float* out = nullptr;
        PIMC_CUDA(nullptr, cudaMalloc(&lines, (size_t)n_lines * kLatLineStrideWords * 8));
        cudaError_t e = cudaMalloc(&out, (size_t)sms * n_lines * sizeof(float));
        if (e == cudaSuccess) e = cudaMemset(lines, 0, (size_t)n_lines * kLatLineStrideWords * 8);
        if (e == cudaSuccess) e = cudaFuncSetAttribute((const void*)lat_l2map_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        void* params[] = {&lines, (void*)&n_lines, &out};
        for (int pass = 0; pass < 2 && e == cudaSuccess; ++pass) {          // the second pass is the measurement
            e = cudaLaunchCooperativeKernel((const void*)lat_l2map_kernel, dim3((unsigned)sms), dim3(32), params, smem, 0);
            if (e == cudaSuccess) e = cudaDeviceSynchronize();
        }
        std::vector<float> lat((size_t)sms * n_lines);
        if (e == cudaSuccess) e = cudaMemcpy(lat.data(), out, lat.size() * sizeof(float), cudaMemcpyDeviceToHost);
        cudaFree(lines); cudaFree(out);
        if (e != cudaSuccess) return fail(nullptr, PIMC_ECUDA, "pimc_latency_selftest: %s", cudaGetErrorString(e));
        // near / far: threshold half way between the 10th and the 90th percentile; SMs grouped by agreement with SM-slot 0's pattern
        std::vector<float> sorted(lat);
        std::sort(sorted.begin(), sorted.end());
        const double thr = 0.5 * ((double)sorted[sorted.size() / 10] + (double)sorted[sorted.size() * 9 / 10]);
        double s_near = 0, s_far = 0; size_t n_near = 0, n_far = 0;
        int group_a = 0;
        for (int b = 0; b < sms; ++b) {
            int agree = 0;
            for (int l = 0; l < n_lines; ++l) {
                const double v = lat[(size_t)b * n_lines + l];
                const bool near = v < thr, near0 = lat[l] < thr;
                if (near) { s_near += v; ++n_near; } else { s_far += v; ++n_far; }
                agree += near == near0;
            }
            group_a += 2 * agree > n_lines;
        }
        out_host[0] = n_near ? s_near / n_near : 0.0;
        out_host[1] = n_far ? s_far / n_far : 0.0;
        out_host[2] = group_a;
        out_host[3] = sms - group_a;
        out_host[4] = (double)n_near / (double)(n_near + n_far);
        return PIMC_OK;
    }
    // one ping-pong measurement: CTAs a <-> b on the line pair at `box`; returns SM clock ticks one way (< 0: CUDA error)
    auto pingpong = [&](int how, int a, int b, unsigned long long* box, long long* out) -> double {
        int rounds = 1010;
        cudaError_t e = cudaMemsetAsync(box, 0, 1024, 0);
        void* params[] = {&how, &a, &b, &rounds, &box, &out};
        if (e == cudaSuccess) e = cudaLaunchCooperativeKernel((const void*)lat_pingpong_kernel, dim3((unsigned)sms), dim3(32), params, smem, 0);
        if (e == cudaSuccess) e = cudaDeviceSynchronize();
        long long cyc = 0;
        if (e == cudaSuccess) e = cudaMemcpy(&cyc, out, sizeof cyc, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) { fail(nullptr, PIMC_ECUDA, "pimc_latency_selftest: %s", cudaGetErrorString(e)); return -1.0; }
        return (double)cyc;
    };
    PIMC_CUDA(nullptr, cudaFuncSetAttribute((const void*)lat_pingpong_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (what <= 5) {
        const int peer = arg <= 0 ? sms - 1 : arg;
        if (peer >= sms) return fail(nullptr, PIMC_EINVAL, "peer must be in [1, SM count)");
        unsigned long long* box = nullptr;
        PIMC_CUDA(nullptr, cudaMalloc(&box, 4096));
        const double v = pingpong(what, 0, peer, box, (long long*)(box + 256));
        cudaFree(box);
        if (v < 0) return PIMC_ECUDA;
        out_host[0] = v;
        return PIMC_OK;
    }
    // what = 6: where the line lives matters.  `arg` line pairs 1 MiB apart (0 = 16, <= 32), plain st.relaxed.gpu, CTA 0 against a
    // handful of peers spread over the grid; the peer with the smallest minimum over the lines shares CTA 0's die, the one with the
    // largest minimum does not (the L2-hit map of what = 0 separates the dies by 35 ticks only: too little to pick pairs from)
    const int n_pairs = arg <= 0 ? 16 : arg;
    if (n_pairs > 32) return fail(nullptr, PIMC_EINVAL, "at most 32 line pairs");
    unsigned long long* big = nullptr;
    PIMC_CUDA(nullptr, cudaMalloc(&big, (size_t)n_pairs << 20));
    long long* outp = nullptr;
    if (cudaMalloc(&outp, 64) != cudaSuccess) { cudaFree(big); return fail(nullptr, PIMC_ENOMEM, "cudaMalloc failed"); }
    const int cand[8] = {1, 2, sms / 4, sms / 2 - 1, sms / 2, 3 * sms / 4, sms - 2, sms - 1};
    double smin = 1e30, smax = 0, cmin = 0, cmax = 0;
    std::vector<double> sv(n_pairs), tv(n_pairs);
    bool ok = true;
    for (int c = 0; c < 8 && ok; ++c) {
        const int peer = cand[c];
        if (peer < 1 || peer >= sms) continue;
        double lo = 1e30, hi = 0;
        for (int k = 0; k < n_pairs && ok; ++k) {
            tv[k] = pingpong(1, 0, peer, big + (size_t)k * (1u << 17), outp);
            ok = tv[k] >= 0;
            lo = std::min(lo, tv[k]); hi = std::max(hi, tv[k]);
        }
        if (lo < smin) { smin = lo; smax = hi; sv = tv; }
        if (lo > cmin) { cmin = lo; cmax = hi; }
    }
    cudaFree(big); cudaFree(outp);
    if (!ok) return PIMC_ECUDA;
    int n_fast = 0;
    for (int k = 0; k < n_pairs; ++k) n_fast += sv[k] < 0.5 * (smin + smax);
    out_host[0] = smin; out_host[1] = smax; out_host[2] = cmin; out_host[3] = cmax; out_host[4] = (double)n_fast / n_pairs;
    return PIMC_OK;
}

const char* pimc_last_error(const pimc_handle* h) { return h ? h->err.c_str() : g_static_error.c_str(); }

int pimc_destroy(pimc_handle* h) {
    if (!h) return PIMC_EINVAL;
    cudaStreamSynchronize(h->stream);
    delete h;
    return PIMC_OK;
}

}  // extern "C"

#endif  // PIMC_PART <= 0

/* pimc.h -- C ABI of libpimc: B200-native (sm_100a) path-integral Monte Carlo hot path.
 *
 * Method: Quinn & Abarbanel, "Data Assimilation using a GPU Accelerated Path Integral Monte Carlo
 * Approach", arXiv 1103.4887.  Citations are /root/reference/PAPER.md:<line> (not present at run time).
 *
 * What is sampled: paths X = {x_0..x_M} (D components per time step) and N_p model parameters p,
 * distributed as exp(-A), with the action (Eq. for A_o, A_d; RK4-map form of the
 * model error named by BASELINE.json's north_star):
 *     A(X,p) = sum_{n=1..M} sum_{l<L} (Rm/2) (y_{n,l} - x_{n,l})^2
 *            + sum_{n=0..M-1} sum_{a<D} (Rf_a/2) ((x_{n+1,a} - x_{n,a}) - g_a(x_n, p; I_n, I_{n+1}))^2
 * where g is the increment of one model step (HH: one classical RK4 step of size dt; LINEAR: A x - x).
 *
 * One "sweep" (Fig. 1): Metropolis update of every even site, then of every odd site
 * (joint Gaussian or uniform proposal of all D components, one accept per site, Eq. 9);
 * then each parameter with non-zero width in sequence (proposals outside
 * [lo,hi] are rejected); then, if enabled, accumulation of running moments and
 * histograms.  All random numbers come from Philox4x32-10 keyed by
 * (seed; site-or-parameter, sweep, chain, stream) so results do not depend on the launch shape.
 *
 * Conventions
 *  - Every function returns PIMC_OK or a negative error; the message of the latest failure can be
 *    read with pimc_last_error().  No C++ exception crosses this boundary.
 *  - Caller-provided device arrays (x, y, I, p, outputs, trace buffers) must be 32-byte aligned: PIMC_EINVAL otherwise.
 *  - "dev" pointers are CUDA device pointers owned by the caller; "host" pointers are ordinary host
 *    memory.  The library copies what it needs into the caller-provided workspace during the call
 *    (asynchronously on `stream`), so inputs may be freed once the stream has passed the call.
 *  - Arrays are row-major and contiguous.  Element type of x, y, I, p, trace arrays = `dtype`
 *    (64: double, 32: float).  Moments are always double, counters unsigned 64-bit.
 *  - All work is enqueued on the ONE `stream` given to pimc_init (a cudaStream_t cast to void*; NULL =
 *    the legacy default stream), for the lifetime of the handle.  Arrays produced or consumed on another stream must be
 *    ordered against it by the caller (event or synchronize).  Nothing synchronises the host except where stated.
 *  - There is no CPU fallback: without a CUDA device every compute call returns PIMC_ECUDA.
 */
#ifndef PIMC_H
#define PIMC_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pimc_handle pimc_handle;

enum { PIMC_OK = 0, PIMC_EINVAL = -1, PIMC_ESTATE = -2, PIMC_ECUDA = -3, PIMC_EUNSUPPORTED = -4, PIMC_ENOMEM = -5 };

/* Models.  LINEAR: D in 1..4, parameters = the D*D map matrix (row-major), g = A x - x.
 * HH: D = 4, x = (V,m,h,n), p = (gNa,gK,gL,ENa,EK,EL,C); tanh kinetics of PAPER.md:256-270 (Eq. 11-14)
 * with Table 1 shifted by -65 mV; needs the injected current I.
 * HH_CLASSIC: as HH, with the classic rate functions da/dt = alpha_a(V)(1-a) - beta_a(V) a of Hodgkin & Huxley (1952),
 * rest at -65 mV: alpha_m = 0.1(V+40)/(1-exp(-(V+40)/10)), beta_m = 4 exp(-(V+65)/18), alpha_h = 0.07 exp(-(V+65)/20),
 * beta_h = 1/(1+exp(-(V+35)/10)), alpha_n = 0.01(V+55)/(1-exp(-(V+55)/10)), beta_n = 0.125 exp(-(V+65)/80)
 * (BASELINE.json says "standard HH"). */
enum { PIMC_MODEL_LINEAR = 0, PIMC_MODEL_HH = 1, PIMC_MODEL_HH_CLASSIC = 2 };
enum { PIMC_PROPOSAL_GAUSSIAN = 0, PIMC_PROPOSAL_UNIFORM = 1 };
/* Sweep engines (same results, different data placement).  GLOBAL: path and cache stay
 * in global memory (L2), threads stride over the tile, neighbour tiles synchronise every half-sweep with
 * release/acquire flags; any tile length.  TILE: each CTA keeps its tile plus h halo sites in shared memory, one
 * (even, odd) site pair per compute thread, halos updated redundantly and exchanged every h half-sweeps as tagged
 * 8-byte packets; needs tile + 2h <= threads_per_cta <= 512 and L = 1 (one observed component).
 * TILE_MC (many chains, PAPER.md:240-242 shared-memory tiles; BASELINE.json config 4 "one CTA-group per chain"): every CTA hosts 2-4
 * independent groups of 128 threads (threads_per_cta = 256, 384 or 512), each with one (chain, tile) pair of at most 256 sites
 * incl. halos resident in shared memory, so that one chain's exchange latency is hidden by the other chains' arithmetic; chains
 * that do not fit at once run in waves (one launch per wave, each running all sweeps of the call).  Hodgkin-Huxley models,
 * RK4-map discretisation, joint updates, L = 1, uniform step sizes, no debug trace, no annealing; halo default 8.
 * AUTO: TILE when it fits; else TILE_MC for two or more chains when it fits; else GLOBAL. */
enum { PIMC_ENGINE_AUTO = 0, PIMC_ENGINE_GLOBAL = 1, PIMC_ENGINE_TILE = 2, PIMC_ENGINE_TILE_MC = 3 };
/* Discretisation of the model-error term between steps n and n+1, (Rf_a/2) r_a^2:
 *  RK4MAP    (default; BASELINE north_star): r = (x_{n+1} - x_n) - g_n, g_n = the increment of one RK4 step from x_n
 *            (LINEAR: g = A x - x); the cache holds g_n, n = 0..M-1.
 *  TRAPEZOID (the paper's own rule, Eq. 7): r = x_{n+1} - x_n - (dt/2)[F(x_{n+1}) + F(x_n)], F the model's
 *            vector field with the current I_n at step n (LINEAR: F(x) = (A x - x)/dt); the cache holds
 *            c_n = (dt/2) F(x_n), n = 0..M (PAPER.md:189, 242 caches F_n).  One right-hand side per proposal instead of
 *            four.  Both engines support both discretisations.  On the TILE engine, and on the GLOBAL engine with one CTA per chain,
 *            the Hodgkin-Huxley models decide ALL parameter moves of a sweep from one reduction of 35 path sums (the cached V term is linear in seven parameter
 *            monomials): same decisions as the per-parameter evaluation, to rounding. */
enum { PIMC_DISC_RK4MAP = 0, PIMC_DISC_TRAPEZOID = 1 };
/* How a site is updated (Fig. 1 proposes all D components together; PAPER.md:226-230 keeps step sizes and
 * acceptance counters per component).  JOINT (default): x'_n = x_n + w o z, one decision per site.  COMPONENTWISE: for
 * a = 0..D-1 in order, x'_{n,a} = x_{n,a} + w_a z_a (the same draw z_a as the joint move) with the other components as they
 * stand, its own Delta-A and decision (accept uniform = words 0,1 of block a of the accept stream); D decisions and D model
 * evaluations per site.  Both engines (TILE: at most 256 threads per CTA).  With the debug trace on, dA_out and acc_out are (n_chains, M+1, D) and xprop_out holds the proposed
 * value of each component. */
enum { PIMC_UPDATE_JOINT = 0, PIMC_UPDATE_COMPONENTWISE = 1 };

/* Number of parameters the model defines (HH: 7, LINEAR: D*D); negative on bad arguments. */
int pimc_model_np(int model, int D);

/* Bytes of device workspace pimc_init needs for this problem (0 on bad arguments). */
size_t pimc_workspace_bytes(int model, int D, int L, int M, int n_chains, int dtype);

/* Create a handle.  model/D/L/M: problem shape (x has M+1 time steps; the first L components are
 * observed, h(x) = x[0:L]).  dt: time step of the RK4 map.  Rm: measurement precision
 * (scalar, R_o of PAPER.md:135).  Rf: host, D model-error precisions (diagonal R_d).
 * p0: host, n_chains*Np initial parameters.  dtype: 64 or 32.  workspace: dev, 256-byte aligned,
 * at least pimc_workspace_bytes(); it is zero-filled here and owned by the caller, who must keep it
 * alive until pimc_destroy.  Errors: PIMC_EINVAL (shape, non-finite dt/Rm/Rf, alignment, size),
 * PIMC_EUNSUPPORTED (D the model does not define), PIMC_ECUDA (no device / CUDA failure). */
int pimc_init(pimc_handle** h, int model, int D, int L, int M, double dt, double Rm, const double* Rf,
              const double* p0, int n_chains, int dtype, void* workspace, size_t workspace_bytes, void* stream);

/* Observations y: dev (n_chains, M+1, L) (y_0 is never used by the action) and injected
 * current I: dev (n_chains, M+1) or NULL (treated as 0).  Rebuilds the step cache if a path is set. */
int pimc_set_data(pimc_handle* h, const void* y, const void* I);

/* Current path x: dev (n_chains, M+1, D).  Copies in and rebuilds the cache g_n = g(x_n,p), n < M
 * ("Calculate and store new RHS").  PIMC_ESTATE before pimc_set_data. */
int pimc_set_path(pimc_handle* h, const void* x);

/* Current parameters p: dev (n_chains, Np).  Copies in and rebuilds the cache. */
int pimc_set_params(pimc_handle* h, const void* p);

/* Copy out the current path (dev (n_chains, M+1, D)) and/or parameters (dev (n_chains, Np)); either may be NULL. */
int pimc_get_path(pimc_handle* h, void* x_out, void* p_out);

/* Copy out the current step cache: dev (n_chains, M, D) for PIMC_DISC_RK4MAP, dev (n_chains, M+1, D) for
 * PIMC_DISC_TRAPEZOID (for cache-coherence checks).  Synchronises the stream. */
int pimc_get_cache(pimc_handle* h, void* g_out);

/* Select the discretisation (PIMC_DISC_*); rebuilds the cache if a path is set.  PIMC_EINVAL on an unknown value. */
int pimc_set_discretisation(pimc_handle* h, int disc);

/* Simulated annealing of the dynamics term (Eq. 10): from the current sweep index on, the model-error
 * weights Rf are multiplied by beta_k = beta0 f^k, f = (1/beta0)^(1/n_cool), k = sweeps since this call, until beta = 1
 * (k >= n_cool); the measurement term is not scaled.  0 < beta0 <= 1; n_cool = 0 switches annealing off.  Both engines
 * carry the schedule (launches that contain a sweep with beta < 1 use the TILE engine's general variant, a few per cent
 * slower than the production one; once the schedule is over the production variant is launched again). */
int pimc_set_annealing(pimc_handle* h, double beta0, long long n_cool);

/* Step-size auto-tuning: from the current sweep index on, every n_skip-th sweep each step size is
 * adjusted, Delta_i <- Delta_i [1 + alpha (N_acc,i / n_skip - f_acc)], N_acc,i = accepted changes of path component
 * i = (n, a) (joint updates: of site n) or of parameter i over the last n_skip sweeps; one step size per (site, component)
 * and per parameter, all starting from the widths of pimc_set_proposal.  enabled = 0 freezes the step sizes as they are
 * (they stay per-site until the next pimc_set_proposal).  Tuning biases the chain: discard its sweeps (the paper tunes during
 * the initialisation phase only).  Both engines tune: the GLOBAL engine adjusts inside its kernel, the TILE engine ends its
 * launches at the adjustment sweeps and adjusts between them (a pimc_sweep call may therefore be several launches); the step
 * sizes are the same bit for bit.  n_skip >= 1, 0 < f_acc < 1 (paper: 0.23), 0 <= alpha < 1 (paper: 0.02). */
int pimc_set_tuning(pimc_handle* h, int enabled, long long n_skip, double f_acc, double alpha);
/* Copy out the step sizes in use: ws_out dev (n_chains, M+1, D) double, wp_out dev (n_chains, Np) double; either may be NULL. */
int pimc_get_widths(pimc_handle* h, double* ws_out, double* wp_out);

/* Select joint or component-wise site updates (PIMC_UPDATE_*).  PIMC_EINVAL on an unknown value. */
int pimc_set_update_mode(pimc_handle* h, int mode);

/* Proposal widths (PAPER.md:188 step (a), 226): w_state host D values >= 0; w_param host Np values >= 0
 * or NULL (= all 0; a parameter with width 0 is frozen and never proposed); kind = PIMC_PROPOSAL_*. */
int pimc_set_proposal(pimc_handle* h, const double* w_state, const double* w_param, int kind);

/* Parameter bounds (uniform prior): host (n_chains, Np) each, lo <= hi.  Default: none. */
int pimc_set_bounds(pimc_handle* h, const double* lo, const double* hi);

/* Moment / histogram accumulation: enabled != 0 accumulates after every n_skip-th sweep,
 * counted from the sweep at which it was (re)enabled or last reset. */
int pimc_set_accum(pimc_handle* h, int enabled, long long n_skip);

/* Zero the running sums and histogram counts and re-centre them on the current path and parameters. */
int pimc_reset_moments(pimc_handle* h);

/* Run n_sweeps sweeps on all chains (asynchronous on the stream; one persistent kernel launch).  The
 * absolute sweep index (part of the RNG counter) continues across calls, so sweep(a)+sweep(b) ==
 * sweep(a+b) bit for bit.  PIMC_ESTATE before set_data/set_path/set_proposal. */
int pimc_sweep(pimc_handle* h, long long n_sweeps, unsigned long long seed);

/* Only the state half-sweeps (rows A2/A3) or only the parameter moves (PAPER.md:199,
 * 209; row A4) of pimc_sweep -- for measuring the two separately.  Same RNG counters as pimc_sweep.  PIMC_ESTATE while
 * step-size tuning is on (the rule needs the acceptance of PROPOSED moves of both classes). */
int pimc_sweep_states_only(pimc_handle* h, long long n_sweeps, unsigned long long seed);
int pimc_sweep_params_only(pimc_handle* h, long long n_sweeps, unsigned long long seed);

/* Moments: out dev double, per chain [mean x (M+1,D), var x (M+1,D), mean p (Np), var p (Np)], chains
 * concatenated; population variance.  n_samples_host (may be NULL) receives the sample count (host
 * bookkeeping, no device sync). */
int pimc_moments(pimc_handle* h, double* out, unsigned long long* n_samples_host);

/* Acceptance counters: acc_out dev u64 (n_chains, 2, D+Np) = accepted, proposed per
 * component class (joint proposals: all D entries equal) and per parameter. */
int pimc_stats(pimc_handle* h, unsigned long long* acc_out);

/* Histograms ("bin counts"): n_sel selections, host arrays: site[i] (>= 0: path site,
 * -1: parameter), comp[i] (component or parameter index), range [lo[i],hi[i]), nbins bins plus an
 * underflow and an overflow bin.  Applies to every chain.  n_sel = 0 disables.  n_sel <= 64. */
int pimc_hist_config(pimc_handle* h, int n_sel, const int* site, const int* comp, const double* lo,
                     const double* hi, int nbins);
/* counts_out: dev u64 (n_chains, n_sel, nbins+2) = under, bins..., over. */
int pimc_hist(pimc_handle* h, unsigned long long* counts_out);

/* Debug trace, filled by the LAST sweep of each later pimc_sweep call (all-NULL disables; no cost then):
 * dA_out dev (n_chains, M+1) per-site Delta-A; acc_out dev u8 (n_chains, M+1) decisions; xprop_out dev
 * (n_chains, M+1, D) proposals or NULL; dA_param dev (n_chains, Np) (NaN = not evaluated: frozen or out of
 * bounds); acc_param dev u8 (n_chains, Np); pprop_out dev (n_chains, Np) proposed parameter values or NULL. */
int pimc_debug_trace(pimc_handle* h, void* dA_out, unsigned char* acc_out, void* xprop_out, void* dA_param,
                     unsigned char* acc_param, void* pprop_out);

/* Launch shape: CTAs per chain (0 = automatic) and threads per CTA (0 = automatic, multiple of 32,
 * <= 1024).  More than one CTA per chain uses a cooperative launch with neighbour hand-off between
 * half-sweeps; PIMC_EINVAL if the grid would not be co-resident. */
int pimc_set_launch(pimc_handle* h, int ctas_per_chain, int threads_per_cta);
/* Report the launch shape that pimc_sweep will use (any pointer may be NULL). */
int pimc_get_launch(pimc_handle* h, int* ctas_per_chain, int* threads_per_cta, int* tile_sites, int* smem_bytes);

/* Choose the sweep engine (PIMC_ENGINE_*) and the halo depth of the TILE engine (-1 = automatic, else even, <= 16:
 * half-sweeps between halo exchanges, row A3).  PIMC_EUNSUPPORTED if the problem does not fit the TILE engine. */
int pimc_set_engine(pimc_handle* h, int engine, int halo);
/* Report the engine and halo depth pimc_sweep will use (any pointer may be NULL). */
int pimc_get_engine(pimc_handle* h, int* engine, int* halo);
/* Optional record of the parameters (Fig. 4 "the evolution of one of the parameters as the MC path update
 * procedure runs"): from now on every ACCUMULATED sweep (pimc_set_accum) writes the chain's parameter vector to record number
 * n_samples of out, dev (n_chains, capacity, Np) of `dtype` elements, owned by the caller; records beyond capacity are dropped;
 * pimc_reset_moments restarts at record 0; out = NULL switches it off.  Written inside the sweep kernels (no extra launch). */
int pimc_param_trace(pimc_handle* h, void* out, long long capacity);

/* Model errors and observation errors of the CURRENT path: eps_out dev (n_chains, M, D),
 * eps_{n,a} = (x_{n+1,a} - x_{n,a}) - g_{n,a} (PIMC_DISC_TRAPEZOID: x_{n+1} - x_n - c_n - c_{n+1}); delta_out dev
 * (n_chains, M+1, L), delta_{n,l} = y_{n,l} - x_{n,l} for n >= 1 and 0 for n = 0 -- the terms of the action, so that
 * A = sum (Rm/2) delta^2 + sum (Rf_a/2) eps^2.  `dtype` elements; either pointer may be NULL. */
int pimc_residuals(pimc_handle* h, void* eps_out, void* delta_out);
/* Running statistics of eps_n and delta_n over the accumulated sweeps ("the means should be zero, the variances should come out as
 * specified by R_o and R_d").  acc: dev double, n_chains x [M*D + M*D + (M+1)*L + (M+1)*L], owned by the caller,
 * zeroed here and by pimc_reset_moments; NULL switches it off.  While it is on, pimc_sweep ends a launch at every accumulated
 * sweep and runs one small kernel on that path (a diagnostic: one extra launch per sample).  pimc_residual_stats: out dev double,
 * same layout = mean eps, var eps, mean delta, var delta (population form, sample count = that of pimc_moments). */
int pimc_set_residual_stats(pimc_handle* h, double* acc);
int pimc_residual_stats(pimc_handle* h, double* out);

/* Tuning knob of the grid-wide Delta-A sum of a parameter move (row A4; TILE engine, more than one CTA per chain): SM clock
 * ticks a CTA waits after publishing its partial before it first polls the other CTAs' packets (default 450; 0 = poll at
 * once).  A packet needs about 1000 ticks from the store to a successful poll; earlier polls only load the L2 slices everybody
 * is waiting on.  Results do not depend on it.  PIMC_EINVAL outside [0, 100000]. */
int pimc_set_exchange(pimc_handle* h, int first_poll_hold_cycles);

/* Synchronise the stream and report whether any inter-CTA hand-off timed out (*fault_host != 0 => PIMC_ECUDA;
 * the chain state is then undefined).  A diagnostic: hand-offs cannot be lost in a co-resident (cooperative) launch. */
int pimc_fault(pimc_handle* h, int* fault_host);

/* The absolute sweep index (part of every RNG counter).  Setting it below the sweep at which accumulation, step-size tuning or
 * annealing was switched on is refused (PIMC_ESTATE): their schedules count sweeps from those origins. */
unsigned long long pimc_sweep_index(const pimc_handle* h);
int pimc_set_sweep_index(pimc_handle* h, unsigned long long t);

/* Number of kernels this handle has launched so far (for bench.py's gpu_launches). */
unsigned long long pimc_launch_count(const pimc_handle* h);

/* End-to-end convenience on HOST buffers (all host, dtype elements except moments): allocates its own
 * device memory, copies y, I (may be NULL), x0, p0 in, runs n_burn sweeps, then n_sweeps sweeps with
 * accumulation every sweep, copies moments_out (host double, layout of pimc_moments) and, if non-NULL,
 * the final path x_out / parameters p_out back, synchronises and frees.  Uses the default stream. */
int pimc_run_host(int model, int D, int L, int M, double dt, double Rm, const double* Rf, int n_chains, int dtype,
                  const void* y, const void* I, const void* x0, const void* p0, const double* w_state,
                  const double* w_param, const double* lo, const double* hi, int proposal_kind, long long n_burn,
                  long long n_sweeps, unsigned long long seed, double* moments_out, void* x_out, void* p_out);

/* The same with a caller-provided device scratch buffer (256-byte aligned, at least pimc_run_host_workspace_bytes(); NULL =
 * allocate as pimc_run_host does), so that repeated calls do not pay cudaMalloc / cudaFree.  Both calls end with the check of
 * pimc_fault: a lost inter-CTA hand-off returns PIMC_ECUDA instead of a result. */
size_t pimc_run_host_workspace_bytes(int model, int D, int L, int M, int n_chains, int dtype);
int pimc_run_host_ws(int model, int D, int L, int M, double dt, double Rm, const double* Rf, int n_chains, int dtype,
                     const void* y, const void* I, const void* x0, const void* p0, const double* w_state,
                     const double* w_param, const double* lo, const double* hi, int proposal_kind, long long n_burn,
                     long long n_sweeps, unsigned long long seed, double* moments_out, void* x_out, void* p_out,
                     void* dev_scratch, size_t dev_scratch_bytes);

/* The same for callers that may not call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it): ALL device memory of the call -- staging copies of y, I, x0, p0, the moments, and the library's workspace (caches,
 * mailboxes, counters) -- is taken from ONE file-scope `static __device__` array of pimc_static_scratch_bytes() = 32 MiB inside
 * libpimc.so (every GPU that loads the library holds it until the process exits).  The call performs no cudaMalloc, cudaFree
 * or allocating library routine.  Arguments, results and error behaviour are those of pimc_run_host (HOST buffers in and out,
 * default stream, synchronises before returning).  Limits: pimc_run_host_workspace_bytes(shape) must not exceed
 * pimc_static_scratch_bytes(), else PIMC_EUNSUPPORTED with the two sizes in pimc_last_error(NULL) -- enough for one chain of
 * M = 32768 in fp64 (28.1 MiB; the headline workload) or any smaller single chain, not for 16 chains of M = 8192 (65 MiB).
 * The array is shared by every call on a device and keeps the last call's contents: each call clears the part it uses before
 * use (what must start at zero: epochs, mailbox tags, counters, moment sums), so calls one after the other are independent,
 * but two calls of this process that overlap on the same GPU (e.g. from two host threads) race on it -- serialise them
 * (other processes have their own copy of the array).  One address per device, looked up once with that device current. */
size_t pimc_static_scratch_bytes(void);
int pimc_run_host_static(int model, int D, int L, int M, double dt, double Rm, const double* Rf, int n_chains, int dtype,
                         const void* y, const void* I, const void* x0, const void* p0, const double* w_state,
                         const double* w_param, const double* lo, const double* hi, int proposal_kind, long long n_burn,
                         long long n_sweeps, unsigned long long seed, double* moments_out, void* x_out, void* p_out);

/* RNG self-test entry (rows A1 / pin P4): fills out (dev u32, n*4) with Philox4x32-10(ctr[i], key), ctrs
 * dev u32 (n,4); and the library's transforms: u_prop dev double n*4 = (w+0.5)2^-32 per word, u_acc dev
 * double n = ((w1:w0 >> 12)+0.5)2^-52, z dev double n*4 = Box-Muller pairs (words 0,1) and (2,3).  Any
 * output may be NULL. */
int pimc_rng_selftest(const unsigned int* ctrs, unsigned long long n, unsigned int key0, unsigned int key1,
                      unsigned int* out, double* u_prop, double* u_acc, double* z, void* stream);

/* Model self-test entry (row A0): g_out dev (n, D) = step increment at x dev (n, D) with parameters p dev (Np),
 * currents I0, I1 dev (n) (NULL = 0), in `dtype` arithmetic. */
int pimc_step_selftest(int model, int D, int dtype, const void* x, const void* p, const void* I0, const void* I1,
                       double dt, unsigned long long n, void* g_out, void* stream);

/* Elementary-function self-test: x dev double (n), out dev double (n,9) = the kernels' own branch-free
 * exp(x) (x clamped to +-700), log|x|, sqrt|x|, sin(min(|x|,7.9)), cos(min(|x|,7.9)), 1/|x|, and the three HH gate rates
 * (a_inf(V) - 0.3)/tau_a(V), a = m, h, n, at V = x (Eq. 12-14; Table 1) as the sweep kernels compute them. */
int pimc_math_selftest(const double* x, unsigned long long n, double* out, void* stream);

/* Roofline denominator probe: runs a register-only chain of independent double-precision FMAs on every SM for
 * roughly `millis` milliseconds and writes the sustained rate in lane-FMA per second (one lane-FMA = one FP64 pipe
 * slot of one thread) to *lane_fma_per_s (host).  Synchronises the device. */
int pimc_fp64_peak_selftest(int millis, double* lane_fma_per_s);

/* Inter-CTA exchange probe (row A4: the grid-wide scalar all-reduce of a parameter move):
 * a cooperative launch of n_ctas CTAs (0 = one per SM) x threads runs `rounds` rounds of { `work` iterations of a register-only
 * FP64 loop with up to 12 % per-CTA jitter, one all-reduce of a per-thread partial }.  mode -1: work only; 0: round 1's flat
 * all-gather (block sum, n_ctas x n_ctas polls, block sum); 1: the two-hop butterfly the sweep kernel uses; 2: block sum, then
 * one warp gathers every block sum; 3: one L2 hop (read the left neighbour's packet).  Host outputs: SM clock ticks per round
 * (after rounds/4 warm-up rounds), the largest |total - exact sum| of the last round over the CTAs, and the number of distinct
 * bit patterns among the CTAs' totals (must be 1: every CTA has to take the same decision).  Synchronises the device. */
int pimc_exchange_selftest(int mode, int n_ctas, int threads, int rounds, int work, double* cycles_per_round_host,
                           double* max_abs_err_host, int* n_distinct_host);

/* Latency probes behind DESIGN.md 6.1a (what one inter-CTA message through L2 is made of).  out: host double[n_out], n_out >= 5.
 *  what = 0: every SM (one CTA per SM, one thread) times dependent chains of ld.relaxed.gpu on each of `arg` lines (0 = 128, <= 256)
 *            4 KB apart, i.e. the cost of an L2 HIT.  The (SM, line) latencies are split at the midpoint of their 10th / 90th
 *            percentile into near and far; out = { mean near ticks, mean far ticks, SMs whose near-pattern agrees with the first
 *            CTA's, the other SMs, fraction of near pairs }: on a two-die part the SMs fall into two equal groups.
 *  what = 1..5: CTA 0 and CTA `arg` (0 = the last) play ping-pong with a tagged 16-byte packet, one reader per line, published with
 *            1 st.relaxed.gpu.v2.u64, 2 two atom.exch.b64, 3 two red.max.u64, 4 st.volatile.v2.u64, 5 st.release.gpu.v2.u64;
 *            out[0] = SM clock ticks one way (store -> the peer's successful poll).
 *  what = 6: the same ping-pong (st.relaxed.gpu) on `arg` line pairs 1 MiB apart (0 = 16, <= 32) between CTA 0 and each of eight peers
 *            spread over the grid; the peer with the smallest minimum over the lines shares CTA 0's die, the one with the largest does
 *            not: out = { same-die min, same-die max, cross-die min, cross-die max one-way ticks, fraction of the line pairs that are
 *            fast for the same-die pair }.  A packet is fast
 *            only when writer, reader and the line's home are on one die; an all-gather always has to cross.
 * Allocates and frees its own device memory, synchronises the device.  PIMC_EINVAL on a bad argument. */
int pimc_latency_selftest(int what, int arg, double* out, int n_out);

const char* pimc_last_error(const pimc_handle* h);   /* h may be NULL: last error of a failed pimc_init / static call */
int pimc_destroy(pimc_handle* h);

#ifdef __cplusplus
}
#endif
#endif /* PIMC_H */

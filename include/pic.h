/* pic.h — C-ABI of the B200-native implicit, adaptive, charge-conserving particle mover
 * (hot path of the fully implicit 1D electrostatic Vlasov-Ampere PIC method of Chen, Chacon &
 * Barnes, arXiv 1111.5295).  Citations: "P:<n>" = /root/reference/PAPER.md line n;
 * "S8(x)" = SURVEY.md section 8(x); "D:<k>" = DESIGN.md section k.
 *
 * The boundary is the paper's: "E down, moments up, particles stay on the GPU".
 * All grid arrays are caller-owned, length n_cells, double precision, and may be HOST or DEVICE
 * pointers (the library asks cudaPointerGetAttributes).  Particle arrays given to pic_init are
 * copied; the handle owns every byte of device state.  All work is enqueued on the CUDA stream
 * given at pic_init; a call that returns data through a HOST pointer synchronises that stream
 * before it returns, a call that only touches DEVICE pointers does not.
 *
 * Every function returns 0 on success or a negative pic_status; nothing throws or aborts across
 * the ABI.  pic_last_error(h) returns a static, NUL-terminated description of the last failure.
 * There is no CPU fallback: without a CUDA device pic_init fails with PIC_ERR_CUDA.
 *
 * Conventions (S8 "Common notation"): periodic domain [0,L), n_cells uniform cells, dx = L/n_cells;
 * face f at x_f = f*dx; cell c spans faces c and (c+1) mod n_cells.  E and jbar live on faces.
 */
#ifndef PAPER_1111_5295_B200_PIC_H
#define PAPER_1111_5295_B200_PIC_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pic_handle pic_handle;

typedef enum pic_status {
  PIC_OK = 0,
  PIC_ERR_ARG = -1,        /* NULL / out-of-range argument                                   */
  PIC_ERR_CUDA = -2,       /* a CUDA runtime call failed (no device, out of memory, fault)   */
  PIC_ERR_PARTICLE = -3,   /* pic_init: a particle has non-finite x or v, or x outside [0,L) */
  PIC_ERR_SUBSTEP_CAP = -4,/* a particle hit max_substeps (A-9); results are still written   */
  PIC_ERR_STATE = -5,      /* call order: pic_residual before pic_set_step, commit before move */
  PIC_ERR_UNSUPPORTED = -6 /* per-visit deposit or (fp32) exact time accounting asked for on a grid
                              too large for shared memory, at pic_init or pic_set_flags; more
                              species than pic_kinetic_energy_noalloc holds                    */
} pic_status;

enum { PIC_FP32 = 0, PIC_FP64 = 1 };   /* arithmetic of the mover kernel (north_star (b))    */
enum { PIC_CN_PICARD = 0,              /* Picard iteration of Eq. 9-10            */
       PIC_CN_DIRECT = 1 };            /* its fixed point, Eq. 11                 */
enum { PIC_STATE_N = 0, PIC_STATE_NP1 = 1 };

/* pic_params.flags */
enum {
  PIC_FLAG_COUNTS = 1,     /* store per-particle n_sub / n_cross (pic_get_counts)             */
  PIC_FLAG_DIAG = 2,       /* count anomalies (kappa cap, clamped roots, ...) in pic_stats     */
  PIC_FLAG_NO_STORE = 4,   /* Krylov calls: skip the state-(n+1) store, only jbar is wanted    */
  PIC_FLAG_VSORT = 8,      /* bin by (cell, |v| class) instead of cell only        */
  PIC_FLAG_NO_DEPOSIT = 32,/* Vlasov-Poisson variant of the mover: no
                              current deposit during the orbit (jbar comes back as 0); the
                              charge density of state n+1 is then pic_rho(PIC_STATE_NP1)      */
  PIC_FLAG_ONE_PER_LANE = 64, /* fp32 only: run the one-particle-per-lane kernel also where the
                              default two-particles-per-lane packed-FP32 kernel (FFMA2) applies;
                              both give bit-identical orbits (A/B timing, tests)               */
  PIC_FLAG_STRIDED = 256,  /* with PIC_FLAG_VSORT: the paper's own particle order (Eq. 15):
                              consecutive particles lie in consecutive CELLS and share a velocity
                              class, instead of sharing a cell (A/B of S8(f) #3; same results)   */
  PIC_FLAG_EXACT_TIME = 128, /* fp32 only: exact accounting of the time used by the sub-steps
                              (fp64 checkpoints of the remaining time, D:5) instead of a plain
                              fp32 `r -= dtau`, whose rounding random-walks to ~ulp(dt) sqrt(n_sub);
                              runs the one-particle-per-lane kernel (the packed two-per-lane one
                              has no such variant); ignored by fp64 handles, whose r is exact
                              enough; PIC_ERR_UNSUPPORTED on grids beyond shared memory          */
  PIC_FLAG_DEPOSIT_PER_VISIT = 16 /* deposit per cell visit with shared fp64 atomics
                              instead of the default end-point form (D:5); same jbar to rounding */
};

typedef struct pic_grid {
  int32_t n_cells;         /* N_g >= 1                                                         */
  int32_t pad_;
  double length;           /* L > 0                                                            */
} pic_grid;

typedef struct pic_species {
  double q_over_m;         /* q/m of the species (a = (q/m) E, Eq. 5)                    */
  double macro_charge;     /* w_q: charge of one macro-particle (sum_p w_q / L = q n0)         */
  int64_t n;               /* number of particles, 0 <= n <= 2^31 - 1 (int32 binning cursors)  */
} pic_species;

typedef struct pic_params {
  double eps_a;            /* absolute tolerance of the sub-step estimator (1e-8 P:277) */
  double eps_r;            /* relative tolerance (0.02)                                 */
  double kappa_max;        /* cap on |a' dtau^2/4| (A-2; 0.5)                                  */
  int32_t max_substeps;    /* per-particle sub-step cap (A-9; 1<<20)                           */
  int32_t picard_max;      /* Picard iteration cap (A-3; 100)                                  */
  int32_t precision;       /* PIC_FP32 | PIC_FP64                                              */
  int32_t cn_mode;         /* PIC_CN_PICARD | PIC_CN_DIRECT                                    */
  uint32_t flags;          /* PIC_FLAG_*                                                       */
  int32_t pad_;
} pic_params;

typedef struct pic_stats { /* totals of the LAST pic_move_accumulate over all species          */
  int64_t n_sub;           /* sub-steps (in-cell + crossing): exact with PIC_FLAG_COUNTS or
                              PIC_FLAG_DIAG; without them the kernel counts in groups of 4
                              rounds and n_sub is an upper bound, < 4 per particle above       */
  int64_t n_cross;         /* crossing sub-steps: exact with PIC_FLAG_COUNTS or PIC_FLAG_DIAG;
                              without them 0 on power-of-two grids (not counted)             */
  int64_t n_picard_it;     /* Picard iterations (PICARD mode)                                  */
  int64_t n_picard_cap;    /* sub-steps whose Picard loop hit picard_max      (DIAG)           */
  int64_t n_kappa_cap;     /* sub-steps limited by the kappa cap              (DIAG)           */
  int64_t n_substep_cap;   /* particles aborted at max_substeps               (always)         */
  int64_t n_neg_disc;      /* crossings with v^2 + 2 a_m d clamped at 0       (DIAG)           */
  int64_t n_clamped_tau;   /* crossings whose dtau_c was clamped to [0,dtau]  (DIAG)           */
  int64_t n_launches;      /* kernels this library launched since pic_init                     */
  double last_move_ms;     /* device time of the mover kernel(s) of the last pic_move_accumulate
                              (CUDA events on the stream; graph-replayed pic_residual calls with
                              host arrays are not timed)                                       */
} pic_stats;

/* pic_init — "pic_init(grid, species, particles)" (north_star (a); S8(b)).
 * x[s], v[s]: n_species pointers to arrays of species[s].n doubles (HOST or DEVICE), positions in
 * [0,L) and velocities.  Validates, computes cell = floor(x/dx) and the in-cell offset
 * xi = x/dx - cell in [0,1] (rounded to the kernel precision), bins particles by cell
 * (north_star (b)) and allocates both state buffers (n and n+1).
 * `stream` is a cudaStream_t (NULL = default stream).  On failure *out is NULL. */
int pic_init(pic_handle** out, const pic_grid* grid, const pic_species* species, int n_species,
             const double* const* x, const double* const* v, const pic_params* params,
             void* stream);

/* pic_move_accumulate — one pass of the hot path a0..a8 (S8(a)) for every species,
 * always starting from state n (particles are enslaved: every residual restarts from x^n, v^n,
 * P:25): field prologue E^{n+1/2} = (E^n + E^{n+1})/2 (north_star), per particle the adaptive
 * sub-step estimate (Eq. 6-8), the Crank-Nicolson move (Eq. 9-11), the
 * cell-crossing truncation (Eq. 12-14) and the linear-spline current deposit
 * (P:210-222), then one reduction per block and the orbit average
 * jbar_f = sum_species w_q (deposit)_f / (dt dx).  Writes state n+1 (scratch until
 * pic_commit) and jbar_out[n_cells].  `tol` is the Picard tolerance (PICARD mode; DIRECT
 * satisfies any tol).  Repeatable: state n is never modified.
 * Returns PIC_ERR_SUBSTEP_CAP if any particle was cut off at max_substeps (checked only when
 * jbar_out is a HOST pointer, since only then the call synchronises; pic_get_stats reports
 * n_substep_cap in every case). */
int pic_move_accumulate(pic_handle* h, const double* E_n, const double* E_np1, double dt,
                        double tol, double* jbar_out);

/* pic_set_step — stores E^n (copied), dt and tol for subsequent pic_residual calls. */
int pic_set_step(pic_handle* h, const double* E_n, double dt, double tol);

/* pic_residual — Ampere residual (north_star; S8(a) a9):
 *   R_f = eps0 (E^{n+1}_f - E^n_f)/dt + jbar_f - <jbar>,  <jbar> = mean over faces, eps0 = 1,
 * with jbar from pic_move_accumulate(E^n, E_np1, dt, tol).  resid_out[n_cells].
 * Returns PIC_ERR_SUBSTEP_CAP (the residual is still written) if any particle was cut off at
 * max_substeps; checked when resid_out is a HOST pointer, as for pic_move_accumulate.
 * With HOST E_np1 and HOST resid_out (the JFNK driver's case) the whole evaluation -- staged copy
 * in, movers, row sum, residual, copy out -- is captured once per (flags, dt, tol) as a CUDA graph
 * and replayed; if `stream` is the legacy default stream the replay runs on a blocking stream of
 * the library's own, which orders with the default stream as usual. */
int pic_residual(pic_handle* h, const double* E_np1, double* resid_out);

/* pic_commit — accept state n+1 of the last pic_move_accumulate as the new state n and re-bin
 * by cell; once per time step, never per residual. */
int pic_commit(pic_handle* h);

/* pic_get_particles — copy one species' state (which = PIC_STATE_N | PIC_STATE_NP1) back in the
 * ORIGINAL particle order of pic_init.  Any output may be NULL.  x = (cell + xi) dx in double;
 * xi is the in-cell offset in cell units exactly as the kernel holds it.  HOST or DEVICE. */
int pic_get_particles(pic_handle* h, int species, int which, double* x, double* v,
                      int32_t* cell, double* xi);

/* pic_get_counts — per-particle sub-step and crossing counts of the last move, original order
 * (needs PIC_FLAG_COUNTS).  HOST or DEVICE. */
int pic_get_counts(pic_handle* h, int species, uint32_t* n_sub, uint32_t* n_cross);

/* pic_count_histogram — histograms over the particles of one species of the per-particle sub-step
 * and crossing counts of the last move (BASELINE.json configs[3]: "sub-step histogram"; needs
 * PIC_FLAG_COUNTS at pic_init and a move made with it).  Bin k counts the particles with
 * k*bin_width <= count < (k+1)*bin_width, the last bin everything above; 1 <= n_bins <= 4096.
 * hist_sub / hist_cross: [n_bins] uint64, HOST or DEVICE, either may be NULL.  Built on the
 * device (the counts never leave it); synchronises the stream. */
int pic_count_histogram(pic_handle* h, int species, uint32_t bin_width, int32_t n_bins,
                        unsigned long long* hist_sub, unsigned long long* hist_cross);

/* pic_get_stats — totals of the last move (synchronises the stream). */
int pic_get_stats(pic_handle* h, pic_stats* out);

/* pic_set_flags — replace pic_params.flags (COUNTS / DIAG / NO_STORE / NO_DEPOSIT /
 * ONE_PER_LANE / DEPOSIT_PER_VISIT / EXACT_TIME) between calls.  PIC_ERR_UNSUPPORTED (flags
 * unchanged) for DEPOSIT_PER_VISIT or fp32 EXACT_TIME on a grid too large for shared memory;
 * PIC_ERR_STATE for COUNTS on a handle created without it (no buffers). */
int pic_set_flags(pic_handle* h, uint32_t flags);

/* pic_kinetic_energy — sum_p w_m v_p^2 / 2 per species (w_m = w_q / (q/m)) of state `which`,
 * reduced on the device in fp64; ke_out[n_species] HOST.  Diagnostic for the energy pin P-9. */
int pic_kinetic_energy(pic_handle* h, int which, double* ke_out);

/* pic_kinetic_energy_noalloc — the same per-species kinetic energy (sum_p w_m v_p^2 / 2, fp64
 * sums; the P-9 energy diagnostic a run evaluates every time step) for host programs that must
 * not allocate GPU memory once their time loop runs: programs whose own pool already holds
 * (nearly) all of the card's memory, so that even the few bytes pic_kinetic_energy cudaMallocs
 * per call may be refused; programs with other streams or handles in flight, which the cudaFree
 * in pic_kinetic_energy would stall (it waits for the whole device); and programs run under a
 * "no allocation after set-up" rule.  This entry point calls no cudaMalloc / cudaFree / allocating
 * routine: its block sums go to a fixed 64 KiB device array that is part of the library image
 * (reserved on every GPU that loads the library, until the process ends).
 *   ke_out[n_species], HOST (the call then synchronises the handle's stream) or DEVICE (it does
 *   not).  which = PIC_STATE_N | PIC_STATE_NP1.
 * Limit: at most PIC_KE_NOALLOC_MAX_SPECIES species per handle (any number of particles);
 * more -> PIC_ERR_UNSUPPORTED with a message, nothing launched.  The handle must live on the
 * CURRENT device (else PIC_ERR_ARG).
 * First call on a device: looks up the array's device address (cudaGetSymbolAddress, which also
 * loads the kernels); make it during set-up, before any stream capture on that device.
 * Sharing: the array is one per GPU, shared by all handles, streams and threads, and keeps the
 * previous call's contents (every slot a call reads it has written first, so nothing needs
 * clearing).  Calls whose GPU work can overlap -- different streams without an ordering between
 * them -- race on it: order them on one stream or with an event.
 * The partial sums are added in a fixed order: same state, same bits, call after call
 * (pic_kinetic_energy's atomics give the same value only up to rounding order). */
enum { PIC_KE_NOALLOC_MAX_SPECIES = 8 };
int pic_kinetic_energy_noalloc(pic_handle* h, int which, double* ke_out);

/* pic_rho — charge density on cell centres, quadratic B-spline (A-10), of state `which`, all
 * species; rho_out[n_cells] HOST or DEVICE.  Used for Gauss-law initialisation (A-13) and the
 * continuity diagnostic; not on the hot path. */
int pic_rho(pic_handle* h, int which, double* rho_out);

/* pic_jfnk_step — one fully implicit time step (north_star (c); S8(f) #1):
 * host fp64 Newton + restarted GMRES on E^{n+1} with the GPU mover as the residual, particles
 * enslaved.  E (HOST, n_cells) holds E^n on entry.  Returns PIC_OK when the step is accepted: E
 * then holds E^{n+1} and the particle state n+1 has been committed (pic_commit) -- the two always
 * change together.  A rejected step changes neither: PIC_ERR_STATE if Newton did not reach
 * rtol/atol within max_newton, PIC_ERR_SUBSTEP_CAP if it converged but orbits of the converged
 * state were cut off at max_substeps (A-9; unlike pic_move_accumulate, whose truncated jbar is
 * still written, a truncated state is never committed); E is then still E^n, the particles are at
 * state n, and the call can be repeated with other settings.  info (may be NULL) receives the
 * iteration counts and residual norms in every case. */
typedef struct pic_jfnk_opts {
  double rtol;             /* nonlinear relative tolerance ||R|| <= rtol ||R_0||                */
  double atol;             /* nonlinear absolute tolerance                                     */
  double fd_eps;           /* finite-difference scale of J w (0 = pick from the precision)     */
  double gmres_rtol;       /* inexact-Newton forcing term                                      */
  int32_t max_newton;
  int32_t gmres_restart;
  int32_t max_gmres;       /* total Krylov iterations per Newton step                          */
  int32_t pad_;
} pic_jfnk_opts;

typedef struct pic_jfnk_info {
  int32_t newton_its;
  int32_t gmres_its;
  int32_t mover_calls;     /* all mover calls of the step                                      */
  int32_t converged;
  double resid0;           /* ||R(E^n)||_2                                                     */
  double resid;            /* final ||R||_2                                                    */
  int32_t mover_calls_resid; /* of which calls of the residual handle (all, without defect corr.) */
  int32_t pad_;
} pic_jfnk_info;

int pic_jfnk_step(pic_handle* h, double* E, double dt, double tol, const pic_jfnk_opts* opts,
                  pic_jfnk_info* info);

/* pic_jfnk_step_dc -- the same step with defect correction (S8(f) #2): the nonlinear
 * residual comes from h_resid (the fp64 mover), the Jacobian-vector products of GMRES from h_jac
 * (the fp32 mover, built from the SAME particles), so the converged E^{n+1} has the accuracy of
 * the fp64 mover while most mover calls run in fp32.  On convergence h_resid is committed and
 * h_jac takes over its state (pic_copy_state). */
int pic_jfnk_step_dc(pic_handle* h_resid, pic_handle* h_jac, double* E, double dt, double tol,
                     const pic_jfnk_opts* opts, pic_jfnk_info* info);

/* pic_copy_state -- make state n of dst a copy of state n of src (same grid, same species and
 * particle counts; precisions may differ: values are converted).  Binning order and original
 * indices are carried over. */
int pic_copy_state(pic_handle* dst, pic_handle* src);

int pic_destroy(pic_handle* h);
const char* pic_last_error(const pic_handle* h);
/* Name of the mover kernel the last pic_move_accumulate launched (static string): "mover2_kernel"
 * (fp32, two particles per lane, packed FP32; csrc/mover2.cuh) or "mover_kernel" (csrc/mover.cuh);
 * "" before the first move.  For bench lines and profiles. */
const char* pic_last_kernel(const pic_handle* h);
/* pic_microbench — the paper's micro-benchmark method on the current device: peak rate
 * of one instruction class in 1e9 thread-operations per second over the whole chip, from a
 * full-occupancy kernel of independent dependent chains timed with CUDA events (divide by n_sm
 * and the SM clock for operations per clock and SM).  which: 0 FFMA, 1 FFMA2 (packed; counts two
 * per thread), 2 FMNMX (ALU pipe), 3 MUFU.RSQ, 4 DFMA, 5 the mix 4 FFMA2 + 4 FMNMX per iteration,
 * 6 the mix 8 FFMA + 4 FMNMX, 7 4 FFMA + 4 FMNMX, 8 2 FFMA2 + 4 FFMA + 4 FMNMX, 9 4 FFMA2 + 2 MUFU.
 * iters: loop length (e.g. 20000).  n_sm may be NULL.  Needs no handle; runs on the default
 * stream and synchronises it. */
int pic_microbench(int which, int iters, double* thread_gops, int* n_sm);

/* pic_debug_bounds — the debug build libpic_b200_check.so (-DPIC_BOUNDS_CHECK=1) checks every
 * shared- and global-memory index its kernels derive from particle data (cell indices, sort
 * keys, scatter destinations, queue positions) and counts the ones out of range (D:7; the pool's
 * compute-sanitizer is closed).  *violations receives that count since the library was loaded
 * (synchronises the device), or -1 from the production build, whose checks compile to nothing.
 * self_test != 0 first provokes exactly one violation, to show that the counter works. */
int pic_debug_bounds(int64_t* violations, int self_test);

/* Library/device identification for logs: fills buf with e.g. "pic_b200 sm_100a ...". */
int pic_version(char* buf, int buflen);

#ifdef __cplusplus
}
#endif
#endif

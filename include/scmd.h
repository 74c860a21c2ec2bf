/*
 * scmd.h -- C ABI of libscmd: the Sutton-Chen molecular-dynamics hot path of
 * arXiv 1210.3559 (Yakubovich et al., "Kinetics of liquid-solid phase transition in
 * large nickel clusters") for one NVIDIA B200 (sm_100a).
 *
 * What the library computes, for a free (non-periodic) cluster of N atoms at r_i:
 *
 *   rho_i = sum_{j != i} (a / r_ij)^m                               Eq. (2)
 *   U     = eps * sum_i [ 1/2 sum_{j != i} (a / r_ij)^n - c sqrt(rho_i) ]   Eq. (1)
 *   F_i   = -dU/dr_i = eps * sum_{j != i} [ n (a/r_ij)^n
 *             - (c m / 2) (rho_i^-1/2 + rho_j^-1/2) (a/r_ij)^m ] (r_i - r_j) / r_ij^2
 *           evaluated as two sweeps over pairs -- first all rho_i, then the forces --
 *           exactly as PAPER.md:127 reduces the many-body term;
 *   velocity-Verlet time stepping, dt in fs ("Verlet integrator with a
 *           time-step of 1 fs"), optionally followed by a velocity-rescale thermostat
 *           (BASELINE.json config 3) or by the paper's Langevin thermostat ("a
 *           Langevin thermostat with a damping constant of 10 ps^-1" = 0.01 fs^-1), discretised as
 *           the exact Ornstein-Uhlenbeck velocity update after the second half kick (see
 *           sc_thermostat).
 *   Parameters for nickel: eps = 1.5707e-2 eV, a = 3.52 A, c = 39.432,
 *           n = 9, m = 6.  The paper runs all pairs with no cutoff; r_cut > 0
 *           selects the cell-list / Verlet-list variant BASELINE.json adds: a pair counts in
 *           rho, energy and force iff r_ij^2 < r_cut^2 (strict, plain truncation).
 *
 * Units: Angstrom, fs, eV, atomic mass unit u, Kelvin.
 *   acceleration = F * SC_ACC / mass,  SC_ACC = 9.648533215665e-3 A fs^-2 per (eV A^-1 u^-1)
 *   KE = 1/2 mass sum |v|^2 / SC_ACC,  T = 2 KE / (kB (3N - 3)),  kB = 8.617333262e-5 eV/K
 *   (T := 0 for N = 1).
 *
 * Pointers: a name starting with d_ is DEVICE memory, h_ is HOST memory.  All arrays are
 * binary64, contiguous, atom-major (N x 3: x0 y0 z0 x1 ...).  The caller owns every buffer
 * it passes, including the workspace, and must keep the workspace alive and untouched
 * until sc_destroy.  The library allocates no device memory of its own.
 *
 * Stream: every call enqueues on the cudaStream_t given to sc_create and returns without
 * waiting, except the calls that return a host scalar or copy to host memory
 * (sc_energy, sc_kinetic, sc_stats, sc_rdf, sc_msd, sc_eval_host, sc_step_host), which synchronise that stream.
 *
 * Errors: every call returns an sc_status; nothing is thrown across the ABI and nothing is
 * printed.  sc_last_error gives a human-readable message for the last failing call on a ctx.
 * There is no CPU fallback: without a CUDA device sc_create returns SC_ERR_CUDA.
 */
#ifndef SCMD_H_
#define SCMD_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sc_ctx sc_ctx; /* opaque; created by sc_create, freed by sc_destroy */

typedef struct {
    int32_t n, m;           /* exponents of Eq. (1)/(2); n > m > 0              */
    double eps, c, a;       /* eV, dimensionless, Angstrom                      */
    double mass;            /* u; BASELINE.json fixes 58.69 for Ni (the paper states none)    */
    double r_cut;           /* Angstrom; <= 0 selects all pairs (the paper's case)            */
} sc_params;

typedef enum {
    SC_OK = 0,
    SC_ERR_INVALID = 1,     /* bad argument: n <= m, m <= 0, N < 1, eps/a/mass <= 0, dt <= 0,
                               skin < 0, NULL pointer, unknown precision / thermostat kind    */
    SC_ERR_CUDA = 2,        /* a CUDA runtime call failed, or no device                        */
    SC_ERR_NOMEM = 3,       /* workspace smaller than sc_workspace_bytes                       */
    SC_ERR_STATE = 4,       /* call needs state that was never set (positions / velocities)   */
    SC_ERR_NONFINITE = 5,   /* a returned scalar is NaN or +-inf (e.g. coincident atoms)       */
    SC_ERR_CAPACITY = 6     /* a neighbour row overflowed its capacity (never truncated)      */
} sc_status;

typedef enum {
    SC_PREC_FP64 = 0,       /* pair arithmetic and accumulation in binary64                    */
    SC_PREC_MIXED = 1       /* pair arithmetic in binary32 on split (hi + lo) coordinates,
                               accumulation in binary64                                        */
} sc_precision;

typedef enum { SC_THERMO_NONE = 0, SC_THERMO_RESCALE = 1, SC_THERMO_LANGEVIN = 2 } sc_thermo_kind;

typedef struct {
    int32_t kind;           /* sc_thermo_kind                                                   */
    double T_start, T_end;  /* K; the bath temperature of step k = 1..nsteps of ONE sc_step call is
                               T_k = T_start + (T_end - T_start) * k / nsteps.
                               RESCALE: after the second half kick, v *= sqrt(T_k / T).
                               LANGEVIN: after the second half kick, v <- c1 v + c2 xi with
                               c1 = exp(-gamma dt), c2 = sqrt((1 - c1^2) kB T_k SC_ACC / mass)    */
    double gamma;           /* 1/fs; Langevin only (10 ps^-1 = 0.01)              */
    uint64_t seed;          /* Langevin only: xi = Box-Muller normals of Philox4x32-10 with key
                               (seed lo, seed hi), counter (atom index in the caller's order,
                               step lo, step hi, 0); the generator step starts at 0 at sc_create,
                               advances by one per Langevin step and can be set with
                               SC_OPT_LANGEVIN_STEP (resume): results do not depend on how a run
                               is split into sc_step calls, on the precision mode's atom order
                               or on the launch configuration                                   */
} sc_thermostat;

/* Runtime options (sc_set_option).  Values are integers; 0 always means "library default". */
typedef enum {
    SC_OPT_ROWS_PER_THREAD = 1,   /* i-atoms held in registers per thread: 1, 2 or 4           */
    SC_OPT_LANES_PER_ROW = 2,     /* lanes of a warp that share one row group: 1,2,4,8,16,32
                                     (list sweeps: lanes per neighbour row, 8, 16 or 32; smaller
                                     values are raised to 8; one-launch step loop: threads of a
                                     row inside one warp)                                        */
    SC_OPT_WARPS_PER_CTA = 3,     /* consumer warps per CTA (they split the j range): 1..8      */
    SC_OPT_PERSISTENT = 4,        /* all pairs: the whole sc_step loop (all nsteps) in ONE cooperative
                                     launch with grid barriers between the phases of a step.  Two
                                     such loops exist: the one-sided one with the records staged in
                                     shared memory (N <= 6144, any thermostat), and the one through
                                     the Newton's-third-law sweeps (NVE and rescale steps, 2048 <= N <= 16384).
                                     0: library default (the first for N <= 2960, the second for NVE and
                                     rescale steps where SC_OPT_NEWTON3 applies and N <= 16384: the measured
                                     crossovers), 1: the first, 2: neither (one launch per sweep
                                     and per integrator stage), 3: never the first.  Off while
                                     sc_profile is on.                                          */
    SC_OPT_ENERGY_EVERY_STEP = 5, /* 1: accumulate pair energy on every step of sc_step          */
    SC_OPT_NEIGHBOUR_CAPACITY = 6,/* K_max entries per row of the Verlet list (cutoff path); rounded
                                     down to a multiple of 32 (at least 32)                      */
    SC_OPT_LANGEVIN_STEP = 7,     /* generator step of the next Langevin update (>= 0)          */
    SC_OPT_CELLS_PER_RADIUS = 8,  /* cutoff path: cell edge = list radius / G, G = 1..4 (default 4);
                                     takes effect at the next list build                         */
    SC_OPT_ATOMS_PER_CTA = 9,     /* cutoff path: consecutive atoms one CTA of the list sweeps
                                     works through (rounded to the warp layout)                  */
    SC_OPT_NEWTON3 = 10,          /* all pairs, either precision, 2048 <= N <= 262144 (the range in which
                                     sc_workspace_bytes includes the ~N^2 / 16 bytes of partial
                                     sums): evaluate every unordered pair once and add its term to
                                     both atoms.  0: library default (on from N = 2961), 1: on,
                                     2: off = the one-sided sweeps                               */
    SC_OPT_CUTOFF_SHIFT = 11,     /* cutoff path: 0 (default) plain truncation, as BASELINE.json's
                                     configs; 1 energy-shifted terms: inside r_cut every pair term
                                     loses its value at the cutoff, (a/r)^k -> (a/r)^k - (a/r_cut)^k
                                     for k = n in Eq. (1) and k = m in Eq. (2), so U is continuous
                                     when a pair crosses r_cut and NVE runs keep their energy; the
                                     force keeps its form, with rho_i the shifted density (DESIGN.md
                                     Q21).  Ignored without a cutoff.                            */
    SC_OPT_NEWTON3_PIECES = 12    /* Newton's-third-law sweeps: how the triangle of unordered pairs is
                                     handed to the CTAs.  0 (default): cut into pieces of equal cost,
                                     one CTA each, one piece per SM;
                                     1..16: that many pieces per SM; -1: a (row block x j segment)
                                     grid with one segment length for all row blocks (rounds 1-2a).
                                     Results are bit-reproducible for a given value, device and N  */
} sc_option;

/* Read-only queries (sc_get_option), beside the sc_option values themselves. */
typedef enum {
    SC_INFO_STEP_PATH = 100,          /* which kernels sc_step / sc_forces run for this context as it is configured now:
                                         0 one-sided all-pairs sweeps, 1 Newton's-third-law all-pairs sweeps,
                                         2 the one-launch step loop (sc_step only; its sc_forces is 0 or 1), 3 cutoff lists */
    SC_INFO_NEIGHBOUR_CAPACITY = 101, /* cutoff path: K_max entries per atom the rows hold now (0 for all pairs)       */
    SC_INFO_NEIGHBOUR_CAPACITY_MAX = 102, /* ... and the largest value the workspace was sized for                       */
    SC_INFO_ONE_LAUNCH = 103          /* 1 if an NVE sc_step call runs all its steps in one cooperative launch as the
                                         context is configured now (SC_OPT_PERSISTENT), else 0                          */
} sc_info;

/* Optional create-time sizing (sc_workspace_bytes_ex / sc_create_ex).  Zero-initialise, then set what is needed;
 * a NULL pointer means all defaults (= sc_workspace_bytes / sc_create). */
typedef struct {
    int32_t neighbour_capacity;   /* cutoff path: K_max entries per atom the neighbour rows are sized for.  0 = default:
                                     1.3 x the fcc number density 4 / a^3 inside the list sphere, which a system denser
                                     than that overflows (SC_ERR_CAPACITY) -- then create the context again with the
                                     max_neighbours sc_stats reported, plus headroom                                    */
    int32_t newton3_storage;      /* all pairs: 0 = carve the ~N^2 / 16 bytes of partial sums of the Newton's-third-law
                                     sweeps where they apply (2048 <= N <= 262144), 2 = never (SC_OPT_NEWTON3 is then
                                     fixed at 2: one-sided sweeps, O(N) workspace)                                      */
    int32_t row_begin, row_end;   /* all pairs over several GPUs: this context is ONE RANK of a row split
                                     and computes / integrates the atoms [row_begin, row_end) only, against all N atoms
                                     (see sc_step_rows).  0, 0 = all rows (one GPU).  Needs r_cut <= 0; the sweeps are the
                                     one-sided ones (a reaction term would have to cross GPUs)                           */
    int32_t reserved[4];          /* must be 0                                                                          */
} sc_create_options;

/* Bytes of device workspace sc_create needs for these arguments (0 on invalid arguments). */
size_t sc_workspace_bytes(const sc_params *params, int64_t n_atoms, int32_t precision, double skin);
size_t sc_workspace_bytes_ex(const sc_params *params, int64_t n_atoms, int32_t precision, double skin,
                             const sc_create_options *options);

/*
 * Create a context for n_atoms atoms.
 *   precision        sc_precision
 *   skin             Angstrom, >= 0; Verlet-list skin for r_cut > 0 (list radius r_cut + skin,
 *                    rebuilt when any atom has moved more than skin / 2 since the last build);
 *                    ignored for r_cut <= 0
 *   d_workspace      device memory, 256-byte aligned, workspace_bytes long, caller-owned
 *   cuda_stream      a cudaStream_t (NULL = legacy default stream)
 *   out              receives the context
 */
sc_status sc_create(const sc_params *params, int64_t n_atoms, int32_t precision, double skin,
                    void *d_workspace, size_t workspace_bytes, void *cuda_stream, sc_ctx **out);
sc_status sc_create_ex(const sc_params *params, int64_t n_atoms, int32_t precision, double skin,
                       const sc_create_options *options, void *d_workspace, size_t workspace_bytes,
                       void *cuda_stream, sc_ctx **out);
sc_status sc_destroy(sc_ctx *ctx);
sc_status sc_set_option(sc_ctx *ctx, int32_t option, int64_t value);
/* Current value of an sc_option (as set, 0 = library default; SC_OPT_LANGEVIN_STEP: the generator step of the
 * next Langevin update, so that a run can be resumed exactly without the caller counting steps) or of an
 * sc_info query.  No device work, no synchronisation. */
sc_status sc_get_option(sc_ctx *ctx, int32_t option, int64_t *value);

/* Copy positions (required) and velocities (d_vel may be NULL: velocities unset) in. */
sc_status sc_set_state(sc_ctx *ctx, const double *d_pos, const double *d_vel);
/* Copy positions / velocities out, in the caller's atom order; either pointer may be NULL. */
sc_status sc_get_state(sc_ctx *ctx, double *d_pos, double *d_vel);

/* First sweep, Eq. (2): d_rho[N]. */
sc_status sc_density(sc_ctx *ctx, double *d_rho);
/* Both sweeps: d_force[N*3] in eV/A.  Also refreshes the cached energy. */
sc_status sc_forces(sc_ctx *ctx, double *d_force);
/* Eq. (1): potential energy in eV of the current positions -> *h_epot.
 * Runs the sweeps if the cached value is stale.  SC_ERR_NONFINITE if not finite. */
sc_status sc_energy(sc_ctx *ctx, double *h_epot);
/* Kinetic energy (eV) and temperature (K) of the current velocities. */
sc_status sc_kinetic(sc_ctx *ctx, double *h_ke, double *h_temperature);
/* nsteps velocity-Verlet steps of dt_fs femtoseconds; thermostat NULL = NVE.
 * SC_ERR_STATE if velocities were never set. */
sc_status sc_step(sc_ctx *ctx, double dt_fs, const sc_thermostat *thermostat, int64_t nsteps);
/*
 * One velocity-Verlet step of a ROW SPLIT over several GPUs (PAPER.md:127's two sweeps each
 * need one exchange).  Every rank holds all N positions and owns the atoms [row_begin, row_end) of its
 * sc_create_options; the exchanges are the caller's (NCCL all-gathers over NVLink on the caller's communicator and
 * stream; the library allocates nothing and knows no communicator).  d_pos_all [N*3] and d_rho_all [N] are the
 * caller's all-atoms arrays.  Per step, on every rank:
 *   phase 0  first half kick + drift of the own atoms; their new positions are written into d_pos_all (own rows only)
 *            -> all-gather d_pos_all
 *   phase 1  all N positions are read from d_pos_all; sweep 1 over the own rows, all j; rho of the own rows is
 *            written into d_rho_all  -> all-gather d_rho_all
 *   phase 2  rho^-1/2 of every atom from d_rho_all; sweep 2 over the own rows (and their share of the pair energy);
 *            second half kick of the own atoms [+ Langevin update, which is local to an atom]
 * sc_energy / sc_kinetic then return THIS RANK'S SHARE of U and KE (sum over its atoms; the temperature is the
 * caller's arithmetic on the all-reduced KE), sc_forces / sc_density / sc_get_state the all-atoms arrays with the own
 * rows current.  Before the first step: sc_set_state (all positions, velocities of at least the own atoms), then
 * phases 1 and 2 with dt_fs = 0 evaluate the forces.  SC_THERMO_RESCALE needs the global temperature between the
 * kick and the scale and is refused here (SC_ERR_INVALID).  dt_fs = 0 in phase 2 skips the kick.
 */
sc_status sc_step_rows(sc_ctx *ctx, int32_t phase, double dt_fs, const sc_thermostat *thermostat, double *d_pos_all,
                       double *d_rho_all);

/* Cutoff-path bookkeeping since sc_create: number of list builds; in-range ordered pairs
 * (r_ij^2 < r_cut^2) at the last force evaluation (N(N-1) for all pairs); longest neighbour
 * row at the last build.  Any pointer may be NULL. */
sc_status sc_stats(sc_ctx *ctx, int64_t *n_rebuilds, int64_t *n_pairs_in_cut, int64_t *max_neighbours);

/*
 * Radial-distribution counts of the central atoms (Eq. (11) g(r) = rho(r) / rho_bar: "the
 * atoms located within 3 A of the cluster center of mass were selected.  For these atoms the RDF was
 * calculated with a distance bin of 0.4 A").  Reference atoms i: |r_i - centre|^2 < r_select^2 (strict);
 * h_counts[b] (host, n_bins entries, 1 <= n_bins <= 4096) = number of ordered pairs (i, j), j != i, with
 * floor(r_ij / bin_width) = b; pairs beyond the last bin are dropped.  The counts are bit-exact (binary64
 * differences, r^2 by fused multiply-add, correctly rounded square root, one multiplication by 1 / bin_width).
 *   h_centre       host, 3 doubles, or NULL = the centre of mass (mean position) computed on the device
 *   h_n_ref        receives the number of reference atoms (may be NULL)
 *   h_centre_used  receives the centre used (host, 3 doubles; may be NULL)
 * The division by n_ref * 4 pi r^2 dr * rho_bar that turns counts into g(r) is left to the caller (the paper
 * does not say which volume defines rho_bar of a finite cluster).  Works on the current positions in any
 * precision mode and with or without a cutoff; synchronises the stream.
 */
sc_status sc_rdf(sc_ctx *ctx, const double *h_centre, double r_select, double bin_width, int32_t n_bins,
                 int64_t *h_counts, int64_t *h_n_ref, double *h_centre_used);

/*
 * Mean-square displacement for the diffusion coefficient D = <dr^2> / (2 z dt), Eq. (12)
 * (PAPER.md:195-199), with the rigid-body fit of PAPER.md:209: "cluster was translated and
 * rotated as a whole in order to minimize the root-mean-square displacement of atoms from a
 * reference structure ... the diffusion coefficient was calculated for all atoms located
 * within 10 A of the cluster center of mass".
 *   d_ref_pos  DEVICE, [N*3] doubles, the reference structure y_i in the caller's atom order
 *              (e.g. an earlier sc_get_state); read only, stays the caller's.
 *   align      0: no fit, displacement x_i - y_i;  1: centroids (equal masses) superposed;
 *              2: centroids superposed and the proper rotation R (det = +1) that minimises
 *              sum_i |R x_i' - y_i'|^2 over ALL atoms (x' = x - centroid of x, likewise y').
 *   r_centre   Angstrom; the average runs over the atoms whose REFERENCE position lies strictly
 *              within r_centre of the reference centroid (Q20); <= 0: every atom.
 *   *h_msd     HOST; mean of |R x_i' - y_i'|^2 over the selected atoms in Angstrom^2 (0 if none
 *              is selected).  D in cm^2/s = 0.1 * msd / (6 * dt_fs) is the caller's arithmetic.
 *   *h_n_sel   HOST, may be NULL; number of selected atoms.
 *   h_rot      HOST, may be NULL; R row-major, 9 doubles (identity for align < 2).  Where the
 *              minimiser is not unique (N = 1, collinear atoms) any minimiser is returned; the
 *              residual is unique.
 * All arithmetic in binary64 in either precision mode; works with and without a cutoff;
 * five small launches, sums in a fixed order (same input -> same bits); synchronises the stream.
 * SC_ERR_STATE without positions, SC_ERR_INVALID for NULL d_ref_pos / h_msd, align outside
 * 0..2 or NaN r_centre, SC_ERR_NONFINITE if the displacement sum is not finite (non-finite
 * reference or positions).
 */
sc_status sc_msd(sc_ctx *ctx, const double *d_ref_pos, double r_centre, int32_t align, double *h_msd,
                 int64_t *h_n_sel, double *h_rot);

/*
 * Host-buffer entry points (the end-to-end path): copies are part of the call.
 * sc_eval_host: upload h_pos[N*3], run both sweeps, download h_force[N*3], h_rho[N] (either
 *   may be NULL) and the potential energy *h_epot (may be NULL).
 * sc_step_host: upload h_pos, h_vel, run nsteps, download both in place, and write
 *   h_scalars[3] = { U, KE, T } of the final state (may be NULL).
 */
sc_status sc_eval_host(sc_ctx *ctx, const double *h_pos, double *h_force, double *h_rho, double *h_epot);
sc_status sc_step_host(sc_ctx *ctx, double *h_pos, double *h_vel, double dt_fs,
                       const sc_thermostat *thermostat, int64_t nsteps, double *h_scalars);

/* Launch accounting: kernels this context has launched since creation. */
sc_status sc_launch_count(sc_ctx *ctx, int64_t *n_launches);
/* Sweep timing for bench.py's roofline line.  After sc_profile(ctx, 1) every force evaluation
 * that runs both sweeps records CUDA events on the ctx stream around each sweep;
 * sc_profile_read synchronises and returns the milliseconds of the most recent one
 * (SC_ERR_STATE if none was recorded). */
sc_status sc_profile(sc_ctx *ctx, int32_t enable);
sc_status sc_profile_read(sc_ctx *ctx, double *h_ms_density, double *h_ms_force);

const char *sc_last_error(const sc_ctx *ctx);
const char *sc_version(void);

/* ---- an entry point that allocates nothing and needs no workspace -----------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it) and so cannot give sc_create a workspace: sweep 1 of the evaluation on its own, all pairs, FP64:
 *     d_rho[i] = sum_{j != i} (a / r_ij)^m                                   Eq. (2)
 *     *d_sum_sqrt_rho = sum_i sqrt(d_rho[i])   (U_emb = -eps c times this, Eq. (1); may be NULL)
 * d_pos: DEVICE, n_atoms x 3 doubles (x, y, z), read only.  d_rho: DEVICE, n_atoms doubles, written.
 * d_sum_sqrt_rho: DEVICE, one double, written (or NULL).  All caller-owned.  cuda_stream: a cudaStream_t (NULL = the
 * default stream); the call enqueues one memset and two kernels on it and returns without waiting.
 * Its scratch -- the packed records and the per-CTA partial sums, which sc_density keeps in the workspace -- lives in a
 * file-scope device array of SC_NOALLOC_SCRATCH_BYTES inside libscmd.so, which every GPU that loads the library holds
 * until the process exits; hence n_atoms <= SC_NOALLOC_MAX_ATOMS, and SC_ERR_NOMEM with a message beyond that.
 * The call makes no cudaMalloc / cudaFree and calls no allocating library routine.  ALL calls share the one array:
 * two calls that overlap on the GPU (different streams or host threads, same device) race on it -- serialise them.
 * Errors: SC_ERR_INVALID (NULL pointer, bad exponents, r_cut > 0: all pairs only, n_atoms < 1), SC_ERR_NOMEM
 * (n_atoms too large), SC_ERR_CUDA; sc_noalloc_last_error gives the calling thread's last message. */
#define SC_NOALLOC_MAX_ATOMS 16384
#define SC_NOALLOC_SCRATCH_BYTES (528 * 1024)
sc_status sc_density_noalloc(const sc_params *params, int64_t n_atoms, const double *d_pos, double *d_rho,
                             double *d_sum_sqrt_rho, void *cuda_stream);
const char *sc_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SCMD_H_ */

/*
 * sc_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU implementation of the Sutton-Chen hot path
 * of arXiv 1210.3559, written from the paper's equations.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call it.  It shares no code, header, table or constant with the CUDA library
 * (paper_1210_3559_b200/csrc); the unit-conversion literals below are retyped here.
 *
 * What it computes (free, non-periodic cluster, all pairs):
 *   Eq. (2)  rho_i = sum_{j != i} (a / r_ij)^m
 *            (the extracted text has the garbled index "i != i"; reading Q2: j != i)
 *   Eq. (1)  U = eps * sum_i [ 1/2 sum_{j != i} (a / r_ij)^n - c sqrt(rho_i) ]
 *   F_i = -dU/dr_i = eps * sum_{j != i} [ n (a/r)^n - (c m / 2)(rho_i^-1/2 + rho_j^-1/2)(a/r)^m ]
 *                          * (r_i - r_j) / r^2
 *            (the paper prints no force formula; this is minus the gradient of Eq. (1),
 *             pinned by central differences in tests/test_oracle_pins.py; two sweeps
 *             as in PAPER.md:127 "first sweep calculating all rho_i ... then ... forces")
 *   velocity-Verlet, dt in fs ("Verlet integrator ... 1 fs"; reading Q3):
 *            v += (dt/2) ACC F/m ; r += dt v ; recompute F ; v += (dt/2) ACC F/m
 *   KE = 1/2 m sum |v|^2 / ACC ;  T = 2 KE / (kB (3N - 3))        (reading Q5)
 *   rescale thermostat after the second half kick: v *= sqrt(T_target / T)   (reading Q6)
 *   Langevin thermostat ("Langevin thermostat with a damping constant of
 *            10 ps^-1"; the discretisation is not stated -- reading Q18): after the second
 *            half kick of step k the exact Ornstein-Uhlenbeck update over dt,
 *              v <- c1 v + c2 xi,  c1 = exp(-gamma dt),  c2 = sqrt((1 - c1^2) kB T_k ACC / m),
 *            T_k the same linear ramp as the rescale thermostat, xi standard normal per
 *            component, drawn from the counter-based generator Philox4x32-10 (Salmon et al.,
 *            SC'11) with key = (seed lo, seed hi) and counter = (atom index, step lo, step hi, 0),
 *            step = step0 + k - 1; words w0..w3 -> u_t = (w_t + 1/2) 2^-32;
 *              xi_x = sqrt(-2 ln u0) cos(2 pi u1), xi_y = sqrt(-2 ln u0) sin(2 pi u1),
 *              xi_z = sqrt(-2 ln u2) cos(2 pi u3)                      (Box-Muller).
 *   cutoff variant (not in the paper; reading Q7): a pair contributes to
 *            rho, pair energy and force iff r2 < r_cut*r_cut, strict, where the decision
 *            value is r2 = fma(dz, dz, fma(dy, dy, dx*dx)) in binary64 with
 *            dx = x_i - x_j etc. in binary64 -- the one place where the precision of an
 *            intermediate is fixed, because floating point decides a set membership.
 *   energy-shifted cutoff (cut_shift = 1, reading Q21): see cut_shift_term below.
 *   rho_i == 0 (atom with no neighbour in range, or N = 1): rho^-1/2 := 0, sqrt(rho) := 0
 *            (reading Q9).  Self term excluded by index (Q11).
 *
 * Powers are repeated multiplication, never pow().  No blocking, no fusion, no Newton's-
 * third-law halving: every ordered pair (i, j) is visited in both sweeps, exactly as the
 * definition reads.  Rows i are independent, so the OpenMP split over i does not change
 * any result.
 *
 * Two builds of this one file:
 *   -DSC_ORACLE_LONG_DOUBLE : pair arithmetic and accumulators in x87 80-bit long double.
 *                             This is the PARITY reference (accurate to ~1e-18 per term).
 *   (default)               : everything in binary64.  This is the build that is TIMED as
 *                             the cpu_baseline.  The two must agree to ~1e-13 (tested).
 *
 * Parity pins: tests/test_oracle_pins.py (closed-form dimer / triangle / tetrahedron /
 * icosahedron / cuboctahedron, mpmath brute force, F = -grad E by central differences,
 * Newton's third law, zero torque, rigid-motion invariance, homogeneity, NVE drift,
 * time reversal, bulk-limit lattice sums, SURVEY.md's independently computed values;
 * Langevin: Philox known-answer vectors, an independent Python restatement of the chain for
 * N = 1, the gamma -> 0 and T = 0 limits, equipartition of free particles).
 * RDF counts: fcc coordination shells 12, 6, 24, 12, 24, 8, 48, the 13-atom icosahedron, the total
 * n_ref (N - 1), numpy brute force.
 * Nothing here is "parity unpinned" except absolute energies against a published
 * number -- the paper prints none.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef SC_ORACLE_LONG_DOUBLE
typedef long double real;
#define R_SQRT sqrtl
#else
typedef double real;
#define R_SQRT sqrt
#endif

/* unit system: Angstrom, fs, eV, u, K.  CODATA-2018 (reading Q4). */
static const double ORACLE_ACC = 9.648533215665e-3;  /* A fs^-2 per (eV A^-1 u^-1) */
static const double ORACLE_KB = 8.617333262e-5;      /* eV / K */

typedef struct {
    int32_t n, m;            /* exponents, n > m > 0 */
    double eps, c, a, mass;  /* eV, -, Angstrom, u */
    double r_cut;            /* Angstrom; <= 0 means all pairs (the paper's case) */
    int32_t cut_shift;       /* with r_cut > 0: 0 plain truncation, 1 energy-shifted terms (reading Q21) */
} oracle_params;

static real ipow(real u, int k) {
    real p = u;
    for (int t = 1; t < k; ++t) p = p * u;
    return p;
}

/* cutoff membership, decided in binary64 exactly as the header states */
static int pair_in_range(const double *pi, const double *pj, double r_cut) {
    if (r_cut <= 0.0) return 1;
    double dx = pi[0] - pj[0], dy = pi[1] - pj[1], dz = pi[2] - pj[2];
    double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    return r2 < r_cut * r_cut;
}

/* Energy-shifted cutoff (reading Q21; not in the paper): inside the cutoff each pair term loses
 * its value at the cutoff, (a/r)^k -> (a/r)^k - (a/r_cut)^k for k = n in Eq. (1) and k = m in Eq. (2), so that
 * U is continuous when a pair crosses r_cut.  Constants drop out of the gradient: the force keeps its form, with
 * rho_i the shifted density.  Returns the constant to subtract (0 without a cutoff or with cut_shift = 0). */
static real cut_shift_term(const oracle_params *p, int k) {
    if (!(p->r_cut > 0.0) || !p->cut_shift) return (real)0;
    return ipow((real)p->a / (real)p->r_cut, k);
}

static real pair_distance(const double *pi, const double *pj, real *d) {
    d[0] = (real)pi[0] - (real)pj[0];
    d[1] = (real)pi[1] - (real)pj[1];
    d[2] = (real)pi[2] - (real)pj[2];
    return R_SQRT(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
}

/* Eq. (2): rho_i for every i (first sweep). */
static void density_real(int64_t N, const double *pos, const oracle_params *p, real *rho) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < N; ++i) {
        real acc = 0;
        const real shift = cut_shift_term(p, p->m);
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            if (!pair_in_range(pos + 3 * i, pos + 3 * j, p->r_cut)) continue;
            real d[3];
            real r = pair_distance(pos + 3 * i, pos + 3 * j, d);
            real u = (real)p->a / r;
            acc += ipow(u, p->m) - shift;
        }
        rho[i] = acc;
    }
}

static real inv_sqrt_or_zero(real rho) { return rho > 0 ? (real)1 / R_SQRT(rho) : (real)0; }

/* second sweep for one row i: force on i and sum_j (a/r)^n */
static void force_row(int64_t N, const double *pos, const oracle_params *p, const real *s,
                      int64_t i, real f[3], real *pair_sum) {
    real fx = 0, fy = 0, fz = 0, ps = 0;
    const real half_cm = (real)p->c * (real)p->m / 2;
    const real shift = cut_shift_term(p, p->n);
    for (int64_t j = 0; j < N; ++j) {
        if (j == i) continue;
        if (!pair_in_range(pos + 3 * i, pos + 3 * j, p->r_cut)) continue;
        real d[3];
        real r = pair_distance(pos + 3 * i, pos + 3 * j, d);
        real u = (real)p->a / r;
        real un = ipow(u, p->n);
        real um = ipow(u, p->m);
        real bracket = (real)p->n * un - half_cm * (s[i] + s[j]) * um;
        real g = (real)p->eps * bracket / (r * r);
        fx += g * d[0];
        fy += g * d[1];
        fz += g * d[2];
        ps += un - shift;
    }
    f[0] = fx; f[1] = fy; f[2] = fz;
    *pair_sum = ps;
}

/* Both sweeps.  Any output pointer may be NULL.  Returns 0, or 1 on allocation failure. */
static int energy_forces_real(int64_t N, const double *pos, const oracle_params *p,
                              real *rho, real *force /*N*3*/, real *e_pair, real *e_emb) {
    real *s = (real *)malloc(sizeof(real) * (size_t)(N > 0 ? N : 1));
    real *ps = (real *)malloc(sizeof(real) * (size_t)(N > 0 ? N : 1));
    if (!s || !ps) { free(s); free(ps); return 1; }
    density_real(N, pos, p, rho);
    for (int64_t i = 0; i < N; ++i) s[i] = inv_sqrt_or_zero(rho[i]);
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < N; ++i) {
        real f[3];
        force_row(N, pos, p, s, i, f, &ps[i]);
        if (force) { force[3 * i] = f[0]; force[3 * i + 1] = f[1]; force[3 * i + 2] = f[2]; }
    }
    real ep = 0, ee = 0;
    for (int64_t i = 0; i < N; ++i) {
        ep += ps[i] / 2;
        ee += (rho[i] > 0 ? R_SQRT(rho[i]) : (real)0);
    }
    if (e_pair) *e_pair = (real)p->eps * ep;
    if (e_emb) *e_emb = -(real)p->eps * (real)p->c * ee;
    free(s); free(ps);
    return 0;
}

static void kinetic_real(int64_t N, const real *vel, double mass, real *ke, real *temp) {
    real acc = 0;
    for (int64_t i = 0; i < 3 * N; ++i) acc += vel[i] * vel[i];
    real k = (real)mass * acc / 2 / (real)ORACLE_ACC;
    *ke = k;
    int64_t ndof = 3 * N - 3;
    *temp = ndof > 0 ? 2 * k / ((real)ORACLE_KB * (real)ndof) : (real)0;
}

/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): ten rounds of
 *   (c0, c1, c2, c3) <- (hi(M1 c2) ^ c1 ^ k0, lo(M1 c2), hi(M0 c0) ^ c3 ^ k1, lo(M0 c0))
 * with the key bumped by the Weyl constants between rounds. */
static void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* the three standard normals of (atom, step) under `seed` -- see the header */
static void langevin_normals(uint64_t seed, uint64_t atom, uint64_t step, double xi[3]) {
    const uint32_t ctr[4] = {(uint32_t)atom, (uint32_t)step, (uint32_t)(step >> 32), 0u};
    const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    uint32_t w[4];
    philox4x32_10(ctr, key, w);
    const double two_pi = 6.283185307179586476925286766559;
    double u0 = ((double)w[0] + 0.5) / 4294967296.0, u1 = ((double)w[1] + 0.5) / 4294967296.0;
    double u2 = ((double)w[2] + 0.5) / 4294967296.0, u3 = ((double)w[3] + 0.5) / 4294967296.0;
    double ra = sqrt(-2.0 * log(u0)), rb = sqrt(-2.0 * log(u2));
    xi[0] = ra * cos(two_pi * u1);
    xi[1] = ra * sin(two_pi * u1);
    xi[2] = rb * cos(two_pi * u3);
}

/* ------------------------------------------------------------------------------------ */
/* exported C entry points (ctypes)                                                       */
/* ------------------------------------------------------------------------------------ */

int oracle_real_bits(void) { return (int)(sizeof(real) * 8); }

int oracle_density(int64_t N, const double *pos, const oracle_params *p, double *rho_out) {
    real *rho = (real *)malloc(sizeof(real) * (size_t)(N > 0 ? N : 1));
    if (!rho) return 1;
    density_real(N, pos, p, rho);
    for (int64_t i = 0; i < N; ++i) rho_out[i] = (double)rho[i];
    free(rho);
    return 0;
}

/* rho_out[N], force_out[N*3], energies[3] = {U, U_pair, U_emb}; any may be NULL */
int oracle_energy_forces(int64_t N, const double *pos, const oracle_params *p,
                         double *rho_out, double *force_out, double *energies) {
    size_t n = (size_t)(N > 0 ? N : 1);
    real *rho = (real *)malloc(sizeof(real) * n);
    real *f = (real *)malloc(sizeof(real) * 3 * n);
    if (!rho || !f) { free(rho); free(f); return 1; }
    real ep, ee;
    int rc = energy_forces_real(N, pos, p, rho, f, &ep, &ee);
    if (!rc) {
        if (rho_out) for (int64_t i = 0; i < N; ++i) rho_out[i] = (double)rho[i];
        if (force_out) for (int64_t i = 0; i < 3 * N; ++i) force_out[i] = (double)f[i];
        if (energies) { energies[0] = (double)(ep + ee); energies[1] = (double)ep; energies[2] = (double)ee; }
    }
    free(rho); free(f);
    return rc;
}

/* Second sweep for a chosen subset of rows, given rho for ALL atoms (from oracle_density).
 * Lets the full-size parity tests check sampled outputs one by one.
 * force_out[nrows*3], pair_sum_out[nrows] (= sum_j (a/r)^n for that row). */
int oracle_forces_rows(int64_t N, const double *pos, const oracle_params *p, const double *rho_all,
                       const int64_t *rows, int64_t nrows, double *force_out, double *pair_sum_out) {
    real *s = (real *)malloc(sizeof(real) * (size_t)(N > 0 ? N : 1));
    if (!s) return 1;
    for (int64_t i = 0; i < N; ++i) s[i] = inv_sqrt_or_zero((real)rho_all[i]);
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t k = 0; k < nrows; ++k) {
        real f[3], ps;
        force_row(N, pos, p, s, rows[k], f, &ps);
        force_out[3 * k] = (double)f[0];
        force_out[3 * k + 1] = (double)f[1];
        force_out[3 * k + 2] = (double)f[2];
        if (pair_sum_out) pair_sum_out[k] = (double)ps;
    }
    free(s);
    return 0;
}

/* First sweep for a chosen subset of rows. */
int oracle_density_rows(int64_t N, const double *pos, const oracle_params *p,
                        const int64_t *rows, int64_t nrows, double *rho_out) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t k = 0; k < nrows; ++k) {
        int64_t i = rows[k];
        real acc = 0;
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            if (!pair_in_range(pos + 3 * i, pos + 3 * j, p->r_cut)) continue;
            real d[3];
            real r = pair_distance(pos + 3 * i, pos + 3 * j, d);
            acc += ipow((real)p->a / r, p->m) - cut_shift_term(p, p->m);
        }
        rho_out[k] = (double)acc;
    }
    return 0;
}

int oracle_kinetic(int64_t N, const double *vel, double mass, double *ke_out, double *temp_out) {
    real *v = (real *)malloc(sizeof(real) * 3 * (size_t)(N > 0 ? N : 1));
    if (!v) return 1;
    for (int64_t i = 0; i < 3 * N; ++i) v[i] = (real)vel[i];
    real ke, t;
    kinetic_real(N, v, mass, &ke, &t);
    *ke_out = (double)ke; *temp_out = (double)t;
    free(v);
    return 0;
}

/* In-range ordered pairs (the cutoff path's "pair interactions"), counted per the header's rule. */
int64_t oracle_count_pairs(int64_t N, const double *pos, double r_cut) {
    int64_t total = 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : total)
    for (int64_t i = 0; i < N; ++i)
        for (int64_t j = 0; j < N; ++j)
            if (j != i && pair_in_range(pos + 3 * i, pos + 3 * j, r_cut)) ++total;
    return total;
}

/*
 * Radial distribution histogram of the central atoms (Eq. (11) and the procedure below
 * it): "the atoms located within 3 A of the cluster center of mass were selected.  For these atoms the RDF
 * was calculated with a distance bin of 0.4 A".  This routine produces the part of g(r) = rho(r) / rho_bar
 * that is a count: counts[b] = number of ordered pairs (i, j), j != i, i a reference atom, with
 * b = floor(r_ij / bin_width), b < n_bins.  Reference atoms: |r_i - centre|^2 < r_select^2, strict.
 *   centre == NULL: the centre of mass (equal masses: the mean position, long double accumulation).
 * Where floating point decides an integer, the precision is fixed (as for the cutoff, reading Q7):
 *   d = x_i - x_j in binary64; r2 = fma(dz, dz, fma(dy, dy, dx*dx)); r = sqrt(r2) (correctly rounded);
 *   b = (int64) floor(r * (1.0 / bin_width)); the selection uses the same r2 form against r_select*r_select.
 * The normalisation to g(r) (division by n_ref * 4 pi r^2 dr * rho_bar; the paper does not say which volume
 * defines rho_bar for a finite cluster -- reading Q19) is arithmetic on these counts and is left to the caller.
 * Returns the number of reference atoms; centre_out (may be NULL) receives the centre used.
 */
int64_t oracle_rdf_counts(int64_t N, const double *pos, const double *centre, double r_select, double bin_width,
                          int64_t n_bins, int64_t *counts, double *centre_out) {
    double c[3];
    if (centre) { c[0] = centre[0]; c[1] = centre[1]; c[2] = centre[2]; }
    else {
        long double s[3] = {0, 0, 0};
        for (int64_t i = 0; i < N; ++i) for (int d = 0; d < 3; ++d) s[d] += pos[3 * i + d];
        for (int d = 0; d < 3; ++d) c[d] = (double)(s[d] / (long double)N);
    }
    if (centre_out) { centre_out[0] = c[0]; centre_out[1] = c[1]; centre_out[2] = c[2]; }
    for (int64_t b = 0; b < n_bins; ++b) counts[b] = 0;
    const double inv_bin = 1.0 / bin_width, rs2 = r_select * r_select;
    int64_t n_ref = 0;
    for (int64_t i = 0; i < N; ++i) {
        const double ex = pos[3 * i] - c[0], ey = pos[3 * i + 1] - c[1], ez = pos[3 * i + 2] - c[2];
        if (!(fma(ez, ez, fma(ey, ey, ex * ex)) < rs2)) continue;
        ++n_ref;
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            const double dx = pos[3 * i] - pos[3 * j], dy = pos[3 * i + 1] - pos[3 * j + 1], dz = pos[3 * i + 2] - pos[3 * j + 2];
            const double r = sqrt(fma(dz, dz, fma(dy, dy, dx * dx)));
            const double fb = floor(r * inv_bin);
            if (fb < (double)n_bins) counts[(int64_t)fb] += 1;
        }
    }
    return n_ref;
}

void oracle_philox4x32_10(const uint32_t *ctr, const uint32_t *key, uint32_t *out) { philox4x32_10(ctr, key, out); }
void oracle_langevin_normals(uint64_t seed, uint64_t atom, uint64_t step, double *xi) { langevin_normals(seed, atom, step, xi); }

/*
 * nsteps of velocity-Verlet from (pos, vel), in place.
 *   thermo_kind 0: NVE.   1: rescale after the second half kick of step k (k = 1..nsteps)
 *   to T_target(k) = T_start + (T_end - T_start) * k / nsteps   (reading Q6).
 *   2: Langevin (reading Q18; gamma in 1/fs, seed, step0 = generator step of this call's first step).
 * Traces (may be NULL), length nsteps + 1, index 0 = initial state:
 *   epot_trace[k], ekin_trace[k] after step k (after the rescale, if any).
 * pos_trace (may be NULL): (nsteps+1) * N * 3 positions.
 * The state is carried in `real` across the whole run.
 */
int oracle_run(int64_t N, double *pos, double *vel, const oracle_params *p, double dt, int64_t nsteps,
               int32_t thermo_kind, double T_start, double T_end, double gamma, uint64_t seed, uint64_t step0,
               double *epot_trace, double *ekin_trace, double *pos_trace) {
    size_t n3 = 3 * (size_t)(N > 0 ? N : 1);
    real *x = (real *)malloc(sizeof(real) * n3);
    real *v = (real *)malloc(sizeof(real) * n3);
    real *f = (real *)malloc(sizeof(real) * n3);
    real *rho = (real *)malloc(sizeof(real) * n3);
    double *xd = (double *)malloc(sizeof(double) * n3);
    if (!x || !v || !f || !rho || !xd) { free(x); free(v); free(f); free(rho); free(xd); return 1; }
    for (int64_t i = 0; i < 3 * N; ++i) { x[i] = (real)pos[i]; v[i] = (real)vel[i]; xd[i] = pos[i]; }
    real ep, ee, ke, temp;
    int rc = energy_forces_real(N, xd, p, rho, f, &ep, &ee);
    if (rc) goto done;
    kinetic_real(N, v, p->mass, &ke, &temp);
    if (epot_trace) epot_trace[0] = (double)(ep + ee);
    if (ekin_trace) ekin_trace[0] = (double)ke;
    if (pos_trace) memcpy(pos_trace, xd, sizeof(double) * 3 * (size_t)N);
    const real half_kick = (real)dt / 2 * (real)ORACLE_ACC / (real)p->mass;
    for (int64_t k = 1; k <= nsteps; ++k) {
        for (int64_t i = 0; i < 3 * N; ++i) v[i] += half_kick * f[i];
        for (int64_t i = 0; i < 3 * N; ++i) x[i] += (real)dt * v[i];
        /* positions are binary64 state at the boundary: round once per step (no-op in the
         * binary64 build) so that the force routine and the next drift see the same x */
        for (int64_t i = 0; i < 3 * N; ++i) { xd[i] = (double)x[i]; x[i] = (real)xd[i]; }
        rc = energy_forces_real(N, xd, p, rho, f, &ep, &ee);
        if (rc) goto done;
        for (int64_t i = 0; i < 3 * N; ++i) v[i] += half_kick * f[i];
        kinetic_real(N, v, p->mass, &ke, &temp);
        if (thermo_kind == 1) {
            real target = (real)T_start + ((real)T_end - (real)T_start) * (real)k / (real)nsteps;
            real lambda = temp > 0 ? R_SQRT(target / temp) : (real)1;
            for (int64_t i = 0; i < 3 * N; ++i) v[i] *= lambda;
            kinetic_real(N, v, p->mass, &ke, &temp);
        } else if (thermo_kind == 2) {
            real target = (real)T_start + ((real)T_end - (real)T_start) * (real)k / (real)nsteps;
            real c1 = (real)exp(-gamma * dt);
            real c2 = R_SQRT(((real)1 - c1 * c1) * (real)ORACLE_KB * target * (real)ORACLE_ACC / (real)p->mass);
            for (int64_t i = 0; i < N; ++i) {
                double xi[3];
                langevin_normals(seed, (uint64_t)i, step0 + (uint64_t)(k - 1), xi);
                for (int d = 0; d < 3; ++d) v[3 * i + d] = c1 * v[3 * i + d] + c2 * (real)xi[d];
            }
            kinetic_real(N, v, p->mass, &ke, &temp);
        }
        if (epot_trace) epot_trace[k] = (double)(ep + ee);
        if (ekin_trace) ekin_trace[k] = (double)ke;
        if (pos_trace) memcpy(pos_trace + (size_t)k * 3 * (size_t)N, xd, sizeof(double) * 3 * (size_t)N);
    }
    for (int64_t i = 0; i < 3 * N; ++i) { pos[i] = (double)x[i]; vel[i] = (double)v[i]; }
done:
    free(x); free(v); free(f); free(rho); free(xd);
    return rc;
}

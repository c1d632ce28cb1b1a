/*
 * sd_oracle.c -- CPU ORACLE for the Stokesian-dynamics mobility product.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or helper with the CUDA path under
 * paper_1205_6333_b200/csrc/ and neither includes the other.
 *
 * What it computes (paper = /root/reference/PAPER.md, Kopp & Hoefling, arXiv:1205.6333):
 *
 *   v_i = mu0 F_i + sum_{j != i} T(r_i - r_j) . F_j            Eq. (7a)
 *   mu0 = 1 / (6 pi eta a)
 *   T(r) = mu0 [ 3a/(4r) (I + rr^) + a^3/(2 r^3) (I - 3 rr^) ] Eq. (7b)
 *   G(r) = 1/(8 pi eta r) (I + rr^)                            Eq. (4),
 *
 * written with rr^ = d d / r^2 (d = r_i - r_j, r = |d|) as
 *
 *   T(d) . F = A(r) F + B(r) (d.F) d
 *
 * The sum is the plain definition: a double loop over all pairs in double precision,
 * every row accumulated in long double.  No blocking, no use of mu_ij = mu_ji, no
 * reordering.  Readings where the paper is silent:
 *   - r < 2a, Rotne-Prager-Yamakawa regularisation (paper silent, PAPER.md:78;
 *     BASELINE.json north_star mandates it):
 *         T = mu0 [ (1 - 9r/(32a)) I + 3/(32 a r) d d ]
 *     r == 2a exactly takes the far branch (both agree there).
 *   - coincident centres (r == 0, j != i): RPY -> mu0 F_j (limit of the overlap branch),
 *     Oseen and unregularised Rotne-Prager -> contribution defined as 0.
 *   - Oseen is evaluated unregularised for every r > 0.
 *   - Euler:  v = M(r) F;  r <- r + dt v.
 *   - Midpoint (north_star; PAPER.md:259 only hints at higher order):
 *         r_h = r + dt/2 M(r) F;   r <- r + dt M(r_h) F.
 *   - forces are inputs (constant during sdo_step).
 *   - periodic box (the *_box entry points; PAPER.md:115 and its footnote 1: "a simulation
 *     box with periodic boundaries and include only hydrodynamic interactions from the
 *     nearest image of each particle"): cubic box of side L; every component of
 *     d = r_i - r_j is replaced by d - L n, n = the integer nearest to d / L, so that
 *     |d_alpha| <= L/2; positions need not lie inside the box; the self pair j == i stays
 *     excluded.  SDO_IMAGE_DEFINITION takes n from C99 remainder() (exact, ties to even).
 *     SDO_IMAGE_F32 / SDO_IMAGE_F64 take the DECISION n the way an fp32 / fp64 evaluation
 *     does (reading B2): n = nearest integer (ties to even) of the exact product
 *     d * inv with inv = 1/L rounded to that precision (and, for F32, d in that product the
 *     fp32 difference of the fp32 positions); the displacement d - L n itself is formed in
 *     double from the exact difference of the stored coordinates.
 *     The variants differ only for pairs within rounding of |d_alpha| = L/2.
 *
 *   - lubrication correction (Eq. 8): see the block comment above
 *     sdo_lubrication; pinned in tests/test_oracle_lub_pins.py.
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): single-sphere Stokes
 * velocity, closed-form two-sphere velocities, continuity and C1-continuity at r = 2a,
 * divergence-freeness, T = (1 + a^2/3 lap) G by finite differences, symmetry,
 * positive definiteness by Cholesky (+ negative controls), invariances, brute-force
 * matrix product, the 517 tau_s four-sphere cycle of PAPER.md:251-253.
 *
 * Positions are never wrapped into the box by sdo_step_box (the nearest-image rule does not
 * need it).
 *
 * Arrays: pos, force, vel are contiguous [N][3] doubles (x, y, z), host memory,
 * caller-owned.  All functions return 0 on success, non-zero on invalid arguments.
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define SDO_TENSOR_RPY 0     /* Eq. (7b) for r >= 2a, RPY overlap form for r < 2a */
#define SDO_TENSOR_OSEEN 1   /* Eq. (4) for every r > 0                          */
#define SDO_TENSOR_RP_FAR 2  /* Eq. (7b) as printed, for every r > 0 (negative control) */

#define SDO_INT_EULER 0
#define SDO_INT_MIDPOINT 1

static const double SDO_PI = 3.14159265358979323846264338327950288;

double sdo_mu0(double a, double eta) { return 1.0 / (6.0 * SDO_PI * eta * a); }

/* Scalar coefficients A(r), B(r) of  T(d).F = A F + B (d.F) d.  Returns 0 if the pair
 * contributes through A, B; 1 if r == 0 (caller applies the coincident-centre reading). */
static int sdo_pair_coef(int tensor, double r, double a, double mu0, double *A, double *B) {
    if (r == 0.0) return 1;
    if (tensor == SDO_TENSOR_OSEEN) {
        /* G = 1/(8 pi eta r)(I + dd/r^2),  1/(8 pi eta) = (3a/4) mu0 */
        *A = mu0 * 3.0 * a / (4.0 * r);
        *B = mu0 * 3.0 * a / (4.0 * r * r * r);
        return 0;
    }
    if (tensor == SDO_TENSOR_RP_FAR || r >= 2.0 * a) {
        /* Eq. (7b): identity part 3a/4r + a^3/2r^3, dyadic part (3a/4r - 3a^3/2r^3)/r^2 */
        *A = mu0 * (3.0 * a / (4.0 * r) + a * a * a / (2.0 * r * r * r));
        *B = mu0 * (3.0 * a / (4.0 * r) - 3.0 * a * a * a / (2.0 * r * r * r)) / (r * r);
        return 0;
    }
    /* RPY, overlapping spheres r < 2a */
    *A = mu0 * (1.0 - 9.0 * r / (32.0 * a));
    *B = mu0 * 3.0 / (32.0 * a * r);
    return 0;
}

#define SDO_IMAGE_DEFINITION 0 /* n from remainder(d, L): the plain definition          */
#define SDO_IMAGE_F32 1        /* n decided as an fp32 evaluation decides it (reading B2) */
#define SDO_IMAGE_F64 2        /* n decided as an fp64 evaluation decides it (reading B2) */

/* nearest integer, ties to even, of the exact value hi + lo (|lo| <= ulp(hi)/2, |hi| < 2^51) */
static double sdo_rint_exact(double hi, double lo) {
    const double t = 2.0 * hi;                                /* exact */
    const int half_integer = (t == floor(t)) && (fmod(t, 2.0) != 0.0); /* hi = k + 1/2 */
    if (half_integer && lo != 0.0) return (lo > 0.0) ? ceil(hi) : floor(hi);
    return nearbyint(hi); /* default rounding mode: to nearest, ties to even */
}

/* Nearest-image displacement of one component (footnote 1).  L <= 0: free space. */
static double sdo_min_image(double xi, double xj, double L, int image) {
    if (!(L > 0.0)) return xi - xj;
    if (image == SDO_IMAGE_F32) {
        const float df = (float)xi - (float)xj;    /* fp32 difference of fp32 positions */
        const float invf = 1.0f / (float)L;        /* 1/L rounded to fp32 */
        const double prod = (double)df * (double)invf; /* 24 x 24 bits: exact in double */
        /* only the DECISION n is taken the fp32 way (reading B2); the displacement is
         * the exact difference of the stored coordinates shifted by n box sides */
        return (xi - xj) - nearbyint(prod) * (double)(float)L;
    }
    const double d = xi - xj;
    if (image == SDO_IMAGE_F64) {
        const double inv = 1.0 / L;
        const double hi = d * inv;
        const double lo = fma(d, inv, -hi);        /* hi + lo = d * inv exactly */
        return d - sdo_rint_exact(hi, lo) * L;
    }
    return remainder(d, L);                        /* d - L * nearest integer to d/L */
}

static int sdo_args_ok(const double *pos, const double *force, long long N, double a, double eta,
                       int tensor) {
    if (!pos || !force || N < 1) return 0;
    if (!(a > 0.0) || !(eta > 0.0) || !isfinite(a) || !isfinite(eta)) return 0;
    if (tensor != SDO_TENSOR_RPY && tensor != SDO_TENSOR_OSEEN && tensor != SDO_TENSOR_RP_FAR)
        return 0;
    return 1;
}

/* One row of Eq. (7a): velocity of particle i. */
static void sdo_row(const double *pos, const double *force, long long N, double a, double mu0,
                    int tensor, double L, int image, long long i, double *v) {
    long double sx, sy, sz;
    const double xi = pos[3 * i + 0], yi = pos[3 * i + 1], zi = pos[3 * i + 2];
    /* self contribution mu_ii = mu0 I */
    sx = (long double)(mu0 * force[3 * i + 0]);
    sy = (long double)(mu0 * force[3 * i + 1]);
    sz = (long double)(mu0 * force[3 * i + 2]);
    for (long long j = 0; j < N; ++j) {
        if (j == i) continue;
        const double dx = sdo_min_image(xi, pos[3 * j + 0], L, image);
        const double dy = sdo_min_image(yi, pos[3 * j + 1], L, image);
        const double dz = sdo_min_image(zi, pos[3 * j + 2], L, image);
        const double fx = force[3 * j + 0], fy = force[3 * j + 1], fz = force[3 * j + 2];
        const double r = sqrt(dx * dx + dy * dy + dz * dz);
        double A, B;
        if (sdo_pair_coef(tensor, r, a, mu0, &A, &B)) {
            if (tensor == SDO_TENSOR_RPY) {
                sx += (long double)(mu0 * fx);
                sy += (long double)(mu0 * fy);
                sz += (long double)(mu0 * fz);
            }
            continue;
        }
        const double dF = dx * fx + dy * fy + dz * fz;
        sx += (long double)(A * fx + B * dF * dx);
        sy += (long double)(A * fy + B * dF * dy);
        sz += (long double)(A * fz + B * dF * dz);
    }
    v[0] = (double)sx;
    v[1] = (double)sy;
    v[2] = (double)sz;
}

static int sdo_box_ok(double L, int image) {
    if (!(L >= 0.0) || !isfinite(L)) return 0;
    return image == SDO_IMAGE_DEFINITION || image == SDO_IMAGE_F32 || image == SDO_IMAGE_F64;
}

/* Velocities of the listed rows only: vel_out[k] = v_{rows[k]}, k < nrows.  L = 0: free space;
 * L > 0: periodic cube of side L, nearest image only (see the header). */
int sdo_apply_rows_box(const double *pos, const double *force, long long N, double a, double eta,
                       int tensor, double L, int image, const long long *rows, long long nrows,
                       double *vel_out) {
    if (!sdo_args_ok(pos, force, N, a, eta, tensor) || !rows || !vel_out || nrows < 0) return 1;
    if (!sdo_box_ok(L, image)) return 1;
    for (long long k = 0; k < nrows; ++k)
        if (rows[k] < 0 || rows[k] >= N) return 1;
    const double mu0 = sdo_mu0(a, eta);
#pragma omp parallel for schedule(dynamic, 8)
    for (long long k = 0; k < nrows; ++k)
        sdo_row(pos, force, N, a, mu0, tensor, L, image, rows[k], vel_out + 3 * k);
    return 0;
}

int sdo_apply_rows(const double *pos, const double *force, long long N, double a, double eta,
                   int tensor, const long long *rows, long long nrows, double *vel_out) {
    return sdo_apply_rows_box(pos, force, N, a, eta, tensor, 0.0, SDO_IMAGE_DEFINITION, rows,
                              nrows, vel_out);
}

/* All rows: vel[i] = v_i, i < N. */
int sdo_apply_box(const double *pos, const double *force, long long N, double a, double eta,
                  int tensor, double L, int image, double *vel) {
    if (!sdo_args_ok(pos, force, N, a, eta, tensor) || !vel || !sdo_box_ok(L, image)) return 1;
    const double mu0 = sdo_mu0(a, eta);
#pragma omp parallel for schedule(dynamic, 8) if (N >= 256)
    for (long long i = 0; i < N; ++i)
        sdo_row(pos, force, N, a, mu0, tensor, L, image, i, vel + 3 * i);
    return 0;
}

int sdo_apply(const double *pos, const double *force, long long N, double a, double eta,
              int tensor, double *vel) {
    return sdo_apply_box(pos, force, N, a, eta, tensor, 0.0, SDO_IMAGE_DEFINITION, vel);
}

/* Dense mobility matrix M[3N][3N], row-major, M[3i+al][3j+be] = (mu_ij)_{al be}. */
int sdo_assemble_box(const double *pos, long long N, double a, double eta, int tensor, double L,
                     int image, double *M) {
    if (!sdo_args_ok(pos, pos, N, a, eta, tensor) || !M || !sdo_box_ok(L, image)) return 1;
    const double mu0 = sdo_mu0(a, eta);
    const long long n3 = 3 * N;
    for (long long i = 0; i < N; ++i) {
        for (long long j = 0; j < N; ++j) {
            double blk[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
            if (i == j) {
                blk[0][0] = blk[1][1] = blk[2][2] = mu0;
            } else {
                double d[3];
                for (int al = 0; al < 3; ++al)
                    d[al] = sdo_min_image(pos[3 * i + al], pos[3 * j + al], L, image);
                const double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
                double A, B;
                if (sdo_pair_coef(tensor, r, a, mu0, &A, &B)) {
                    if (tensor == SDO_TENSOR_RPY) blk[0][0] = blk[1][1] = blk[2][2] = mu0;
                } else {
                    for (int al = 0; al < 3; ++al)
                        for (int be = 0; be < 3; ++be)
                            blk[al][be] = (al == be ? A : 0.0) + B * d[al] * d[be];
                }
            }
            for (int al = 0; al < 3; ++al)
                for (int be = 0; be < 3; ++be) M[(3 * i + al) * n3 + (3 * j + be)] = blk[al][be];
        }
    }
    return 0;
}

int sdo_assemble(const double *pos, long long N, double a, double eta, int tensor, double *M) {
    return sdo_assemble_box(pos, N, a, eta, tensor, 0.0, SDO_IMAGE_DEFINITION, M);
}

/* Explicit integration with constant forces.  pos is updated in place.
 * If traj != NULL, the positions after steps rec_stride, 2 rec_stride, ... are appended to
 * traj ([n_steps / rec_stride][N][3]).  vel_last (optional) receives the velocities of the
 * last product evaluated (Euler: M(r_n)F of the last step; midpoint: M(r_h)F). */
int sdo_step_box(double *pos, const double *force, long long N, double a, double eta, int tensor,
                 double L, int image, double dt, long long n_steps, int integrator, double *traj,
                 long long rec_stride, double *vel_last) {
    if (!sdo_args_ok(pos, force, N, a, eta, tensor) || !isfinite(dt) || n_steps < 0) return 1;
    if (!sdo_box_ok(L, image)) return 1;
    if (integrator != SDO_INT_EULER && integrator != SDO_INT_MIDPOINT) return 1;
    if (traj && rec_stride < 1) return 1;
    double *v = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    double *ph = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    if (!v || !ph) {
        free(v);
        free(ph);
        return 2;
    }
    long long nrec = 0;
    for (long long s = 0; s < n_steps; ++s) {
        sdo_apply_box(pos, force, N, a, eta, tensor, L, image, v);
        if (integrator == SDO_INT_EULER) {
            for (long long k = 0; k < 3 * N; ++k) pos[k] = pos[k] + dt * v[k];
        } else {
            for (long long k = 0; k < 3 * N; ++k) ph[k] = pos[k] + 0.5 * dt * v[k];
            sdo_apply_box(ph, force, N, a, eta, tensor, L, image, v);
            for (long long k = 0; k < 3 * N; ++k) pos[k] = pos[k] + dt * v[k];
        }
        if (traj && (s + 1) % rec_stride == 0) {
            memcpy(traj + (size_t)nrec * 3 * (size_t)N, pos, sizeof(double) * 3 * (size_t)N);
            ++nrec;
        }
    }
    if (vel_last && n_steps > 0) memcpy(vel_last, v, sizeof(double) * 3 * (size_t)N);
    free(v);
    free(ph);
    return 0;
}

int sdo_step(double *pos, const double *force, long long N, double a, double eta, int tensor,
             double dt, long long n_steps, int integrator, double *traj, long long rec_stride,
             double *vel_last) {
    return sdo_step_box(pos, force, N, a, eta, tensor, 0.0, SDO_IMAGE_DEFINITION, dt, n_steps,
                        integrator, traj, rec_stride, vel_last);
}

/* ---- lubrication correction (Eq. 8) --------------------
 *
 *   mu0 f_sing(r_ij) = [ 1/(4 s) - (9/40) ln s ] rr^ - (1/6) ln s (I - rr^),   s = r_ij / a - 2
 *   C_i = sum'_j f_sing(r_ij) . (v_i - v_j)         (the term subtracted from F_i in step 2 of
 *                                                    the paper's loop)
 * Readings (C1-C4): the primed sum runs over j != i with r_ij < 3a ("we truncate ad hoc
 * at s = 1 or r = 3a"); ln is the natural logarithm; s is clamped from below at SDO_LUB_SMIN (the
 * paper never lets spheres touch; Eq. 8 diverges at s = 0 and is undefined for s < 0); periodic
 * box as in sdo_apply_box.  decide_f32 != 0 takes the DECISION r < 3a the way the fp32 kernels
 * do: on r^2 = fma(dz,dz,fma(dy,dy,dx*dx)) evaluated in float on float displacements, against
 * (float)(9 a^2); the term itself is always evaluated in double.
 */
#define SDO_LUB_SMIN 1.0e-3

static void sdo_lub_row(const double *pos, const double *vel, long long N, double a, double mu0,
                        double L, int image, int decide_f32, long long i, double *c) {
    long double sx = 0.0L, sy = 0.0L, sz = 0.0L;
    for (long long j = 0; j < N; ++j) {
        if (j == i) continue;
        const double dx = sdo_min_image(pos[3 * i + 0], pos[3 * j + 0], L, image);
        const double dy = sdo_min_image(pos[3 * i + 1], pos[3 * j + 1], L, image);
        const double dz = sdo_min_image(pos[3 * i + 2], pos[3 * j + 2], L, image);
        const double r2 = dx * dx + dy * dy + dz * dz;
        int inside;
        if (decide_f32) {
            const float fx = (float)dx, fy = (float)dy, fz = (float)dz;
            inside = fmaf(fz, fz, fmaf(fy, fy, fx * fx)) < (float)(9.0 * a * a);
        } else {
            inside = r2 < 9.0 * a * a;
        }
        if (!inside || r2 == 0.0) continue;
        const double r = sqrt(r2);
        double s = r / a - 2.0;
        if (s < SDO_LUB_SMIN) s = SDO_LUB_SMIN;
        const double ls = log(s);
        const double par = (1.0 / (4.0 * s) - 9.0 / 40.0 * ls) / mu0; /* along rr^      */
        const double per = (-ls / 6.0) / mu0;                         /* along I - rr^  */
        const double wx = vel[3 * i + 0] - vel[3 * j + 0];
        const double wy = vel[3 * i + 1] - vel[3 * j + 1];
        const double wz = vel[3 * i + 2] - vel[3 * j + 2];
        const double rw = (dx * wx + dy * wy + dz * wz) / r2;         /* (r^ . w) / r   */
        sx += (long double)(per * wx + (par - per) * rw * dx);
        sy += (long double)(per * wy + (par - per) * rw * dy);
        sz += (long double)(per * wz + (par - per) * rw * dz);
    }
    c[0] = (double)sx;
    c[1] = (double)sy;
    c[2] = (double)sz;
}

/* corr[i] = C_i for all i.  vel: [N][3] velocities of the previous step. */
int sdo_lubrication(const double *pos, const double *vel, long long N, double a, double eta,
                    double L, int image, int decide_f32, double *corr) {
    if (!sdo_args_ok(pos, vel, N, a, eta, SDO_TENSOR_RPY) || !corr || !sdo_box_ok(L, image)) return 1;
    const double mu0 = sdo_mu0(a, eta);
#pragma omp parallel for schedule(dynamic, 8) if (N >= 256)
    for (long long i = 0; i < N; ++i)
        sdo_lub_row(pos, vel, N, a, mu0, L, image, decide_f32, i, corr + 3 * i);
    return 0;
}

/* The paper's loop with the lubrication-corrected forces, constant external
 * forces fext:  F = fext - C(r, v_prev);  v = M(r) F;  Euler: r <- r + dt v.  Midpoint: both
 * stages correct the forces with the velocities of the product evaluated last.  vel: in = the
 * velocities "of the previous step" (zeros for a cold start), out = those of the last product. */
int sdo_step_lub(double *pos, double *vel, const double *fext, long long N, double a, double eta,
                 int tensor, double L, int image, int decide_f32, double dt, long long n_steps,
                 int integrator) {
    if (!sdo_args_ok(pos, fext, N, a, eta, tensor) || !vel || !isfinite(dt) || n_steps < 0) return 1;
    if (!sdo_box_ok(L, image)) return 1;
    if (integrator != SDO_INT_EULER && integrator != SDO_INT_MIDPOINT) return 1;
    const size_t n3 = 3 * (size_t)N;
    double *f = (double *)malloc(sizeof(double) * n3);
    double *c = (double *)malloc(sizeof(double) * n3);
    double *ph = (double *)malloc(sizeof(double) * n3);
    if (!f || !c || !ph) {
        free(f); free(c); free(ph);
        return 2;
    }
    for (long long s = 0; s < n_steps; ++s) {
        sdo_lubrication(pos, vel, N, a, eta, L, image, decide_f32, c);
        for (size_t k = 0; k < n3; ++k) f[k] = fext[k] - c[k];
        sdo_apply_box(pos, f, N, a, eta, tensor, L, image, vel);
        if (integrator == SDO_INT_EULER) {
            for (size_t k = 0; k < n3; ++k) pos[k] = pos[k] + dt * vel[k];
        } else {
            for (size_t k = 0; k < n3; ++k) ph[k] = pos[k] + 0.5 * dt * vel[k];
            sdo_lubrication(ph, vel, N, a, eta, L, image, decide_f32, c);
            for (size_t k = 0; k < n3; ++k) f[k] = fext[k] - c[k];
            sdo_apply_box(ph, f, N, a, eta, tensor, L, image, vel);
            for (size_t k = 0; k < n3; ++k) pos[k] = pos[k] + dt * vel[k];
        }
    }
    free(f); free(c); free(ph);
    return 0;
}

int sdo_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void sdo_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

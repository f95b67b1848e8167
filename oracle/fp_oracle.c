/*
 * fp_oracle.c -- plain, slow, obviously-correct CPU oracle for the cubic Fokker-Planck closure hot path
 * of arxiv/paper_2606_15622.  TEST INFRASTRUCTURE ONLY: only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call this file.  It shares no code,
 * headers, tables or helpers with the CUDA path (paper_2606_15622_b200/csrc) and neither includes the other.
 *
 * Arithmetic: fp64 everywhere on the fp32 inputs, EXCEPT where a floating-point value decides an integer or
 * a stored position (cell index S1, streaming/wall positions S7): there the fp32 operation sequence is part
 * of the definition and both sides evaluate exactly it.  Compile with -O2 -ffp-contract=off.
 *
 * Every function cites the PAPER.md passage it follows (line numbers of /root/reference/PAPER.md) and,
 * where the paper is silent or garbled, the reading recorded in DESIGN.md "Readings" (R-numbers; they are
 * the S-numbers of SURVEY.md section 8(c)).
 *
 * Parity pins (tests/test_oracle_*.py): moments -- hand values, Maxwellian closed forms, Galilean invariance;
 * exact closure -- Langevin special case (Eq. 4), linearised Grad-13 closed form, substitution of the solved
 * coefficients into the relaxation constraints evaluated from particles (bypasses the matrix), residual,
 * brute-force Cramer, axis-permutation and scaling symmetries, Table 1 entries as printed; MLP -- hand cases,
 * parameter counts, independent numpy forward; Philox -- Random123 known-answer vectors and
 * numpy's Philox bit generator; update -- Eq. 15 identity, noise-off Langevin decay, conservation, OU
 * stationarity, the drift N_i recovered from the OUTPUT velocities against Eq. 14 typed out in numpy and against
 * the relaxation identities the exact closure imposes (<N_i c_j + N_j c_i> = 0, <N_i c^2 + 2 c_i c.N> = 5 h_i/(3 tau)),
 * an N = 2 cell is updated; walls -- half-range Maxwellian moments on the lid (y-wall) and on both Couette plates
 * (x-walls, distinct tangential wall speeds), the freestream reservoir against the analytic moments of the flux-weighted
 * drifting half-range Maxwellian at two speed ratios; diagnostics -- hand values on octahedral ensembles, numpy
 * slogdet, rotation invariance, Maxwellian limits, N = 3 cells whose determinant rounds positive.
 * Parity unpinned (no independent source exists): the value of eps^2 (R2-e), the low-count /
 * singular-cell policy (R3-c), the 16-feature definitions (R4), the wall re-emission details (R7), the reservoir's
 * algorithm (R11: the law it samples is pinned, that the paper's code does the same is not) and the no-history rule of
 * the under-relaxation (R12), each as compared with the paper's own runs.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_PI 3.14159265358979323846

/* The per-cell (moments, closures, update) and per-particle (streaming) loops carry `#pragma omp parallel for`: iterations
 * are independent and write disjoint outputs, so the result does not depend on the thread count.  The pragmas are
 * inert unless the file is compiled with -fopenmp (oracle.py does); orc_set_threads picks the count (bench.py times
 * one thread and all cores). */
#ifdef _OPENMP
#include <omp.h>
void orc_set_threads(int n) { omp_set_num_threads(n > 0 ? n : omp_get_num_procs()); }
int orc_max_threads(void) { return omp_get_max_threads(); }
#else
void orc_set_threads(int n) { (void)n; }
int orc_max_threads(void) { return 1; }
#endif

/* per-cell flag bits (interface constants, stated in include/fpcl.h as FP_FLAG_*) */
#define ORC_FLAG_EMPTY     1u   /* N == 0                                            */
#define ORC_FLAG_LOWCOUNT  2u   /* N < min_count: Langevin fallback (R3-c)           */
#define ORC_FLAG_SINGULAR  4u   /* theta<=0, tiny pivot or non-finite: Langevin      */
#define ORC_FLAG_ILLCOND   8u   /* kappa_1 >= 1e8, solution kept                     */
#define ORC_FLAG_ALPHA    16u   /* alpha^2 non-finite or < 1e-6: alpha := 1 (R5.3)   */
#define ORC_FLAG_SKIPPED  32u   /* update skipped: N < 2 or theta <= 0 (R5)          */
#define ORC_FLAG_NONFINITE 64u  /* a non-finite value was produced and replaced      */

/* ------------------------------------------------------------------------------------------------
 * S1 / R1 -- cell index, stable sort, counts.  PAPER.md:215 (sort_and_calc_moments), :728 ("shared sorting").
 * The paper gives no formula.  Reading R1: ix = clamp(floorf((x - x0) * inv_dx), 0, nx-1) evaluated in fp32
 * (subtract, then multiply; inv_dx = 1.0f/dx computed once in fp32), key = iy*nx + ix.  NaN maps to 0.
 * ------------------------------------------------------------------------------------------------ */
static int32_t orc_axis_index(float p, float p0, float inv_d, int32_t n)
{
    float f = (p - p0) * inv_d;          /* fp32, two roundings; -ffp-contract=off keeps it that way */
    float t = floorf(f);
    if (!(t >= 0.0f)) return 0;          /* negatives and NaN */
    if (t >= (float)n) return n - 1;
    return (int32_t)t;
}

void orc_cell_index(int64_t np, const float *x, const float *y, int32_t nx, int32_t ny,
                    float x0, float y0, float dx, float dy, int32_t *key)
{
    float inv_dx = 1.0f / dx, inv_dy = 1.0f / dy;
    for (int64_t p = 0; p < np; ++p) {
        int32_t ix = orc_axis_index(x[p], x0, inv_dx, nx);
        int32_t iy = (ny > 1) ? orc_axis_index(y[p], y0, inv_dy, ny) : 0;
        key[p] = iy * nx + ix;
    }
}

/* Stable sort by key: equal keys keep input order (R1: the only reading under which "sort order" is unique).
 * Written as the definition of a stable counting sort: count, exclusive prefix, place in input order.
 * cell_start[k] = #particles with key < k, cell_start[ncell] = np; perm[k] = input index now at position k. */
void orc_sort_by_key(int64_t np, const int32_t *key, int32_t ncell, int32_t *cell_start, uint32_t *perm)
{
    int64_t *cursor = (int64_t *)calloc((size_t)ncell + 1, sizeof(int64_t));
    for (int64_t p = 0; p < np; ++p) cursor[key[p] + 1] += 1;
    for (int32_t c = 0; c < ncell; ++c) cursor[c + 1] += cursor[c];
    for (int32_t c = 0; c <= ncell; ++c) cell_start[c] = (int32_t)cursor[c];
    for (int64_t p = 0; p < np; ++p) { perm[cursor[key[p]]] = (uint32_t)p; cursor[key[p]] += 1; }
    free(cursor);
}

/* ------------------------------------------------------------------------------------------------
 * S0 / R0 -- per-cell velocity moments.  PAPER.md:124 (u^(p)_{i1..in} = int |v'|^p v'_i1..v'_in f dV),
 * :215-216 (M1-M5), :243 (LITE skips M3..M5), :415 (theta = <c_k c_k>/3), :181 (<.> is the plain mean, 1/N).
 * Two passes in fp64 over the cell's fp32 velocities.
 * FULL record (29): N, U1..3, P11,P12,P13,P22,P23,P33, t111,t112,t113,t122,t123,t133,t222,t223,t233,t333,
 *                   F11,F12,F13,F22,F23,F33 (F_ij = <c^2 c_i c_j>), g1,g2,g3 (g_i = <c^4 c_i>).
 * LITE record (13): N, U1..3, P(6), h1,h2,h3 (h_i = <c^2 c_i>).
 * Empty cell: all zeros.
 * ------------------------------------------------------------------------------------------------ */
void orc_cell_moments(const float *vx, const float *vy, const float *vz, const int32_t *cell_start,
                      int32_t ncell, int32_t mode, double *mom)
{
    const int stride = mode ? 29 : 13;
#pragma omp parallel for schedule(dynamic, 64)
    for (int32_t cell = 0; cell < ncell; ++cell) {
        double *m = mom + (size_t)cell * stride;
        for (int k = 0; k < stride; ++k) m[k] = 0.0;
        int64_t s = cell_start[cell], e = cell_start[cell + 1];
        int64_t n = e - s;
        if (n <= 0) continue;
        double U[3] = {0, 0, 0};
        for (int64_t p = s; p < e; ++p) { U[0] += vx[p]; U[1] += vy[p]; U[2] += vz[p]; }
        for (int i = 0; i < 3; ++i) U[i] /= (double)n;
        double P[6] = {0}, t[10] = {0}, F[6] = {0}, g[3] = {0}, h[3] = {0};
        for (int64_t p = s; p < e; ++p) {
            double c[3] = {(double)vx[p] - U[0], (double)vy[p] - U[1], (double)vz[p] - U[2]};
            double c2 = c[0] * c[0] + c[1] * c[1] + c[2] * c[2];
            int a = 0, b = 0;
            for (int i = 0; i < 3; ++i)
                for (int j = i; j < 3; ++j) {
                    P[a] += c[i] * c[j];
                    F[a] += c2 * c[i] * c[j];
                    ++a;
                    for (int k = j; k < 3; ++k) t[b++] += c[i] * c[j] * c[k];
                }
            for (int i = 0; i < 3; ++i) { h[i] += c2 * c[i]; g[i] += c2 * c2 * c[i]; }
        }
        double inv = 1.0 / (double)n;
        m[0] = (double)n; m[1] = U[0]; m[2] = U[1]; m[3] = U[2];
        for (int k = 0; k < 6; ++k) m[4 + k] = P[k] * inv;
        if (mode) {
            for (int k = 0; k < 10; ++k) m[10 + k] = t[k] * inv;
            for (int k = 0; k < 6; ++k) m[20 + k] = F[k] * inv;
            for (int k = 0; k < 3; ++k) m[26 + k] = g[k] * inv;
        } else {
            for (int k = 0; k < 3; ++k) m[10 + k] = h[k] * inv;
        }
    }
}

/* helpers to read a record: symmetric index maps.  sym2: (i,j)->0..5 in order 11,12,13,22,23,33;
 * sym3: (i,j,k)->0..9 in order 111,112,113,122,123,133,222,223,233,333. */
static int sym2(int i, int j)
{
    if (i > j) { int s = i; i = j; j = s; }
    static const int map[3][3] = {{0, 1, 2}, {-1, 3, 4}, {-1, -1, 5}};
    return map[i][j];
}
static int sym3(int i, int j, int k)
{
    int a[3] = {i, j, k};
    for (int p = 0; p < 2; ++p) for (int q = 0; q < 2 - p; ++q) if (a[q] > a[q + 1]) { int s = a[q]; a[q] = a[q + 1]; a[q + 1] = s; }
    static const int map[3][3][3] = {
        {{0, 1, 2}, {-1, 3, 4}, {-1, -1, 5}},
        {{-1, -1, -1}, {-1, 6, 7}, {-1, -1, 8}},
        {{-1, -1, -1}, {-1, -1, -1}, {-1, -1, 9}}};
    return map[a[0]][a[1]][a[2]];
}

/* h_i = <c^2 c_i> from either record layout: LITE stores it, FULL gives it as t_ikk (R0). */
static void orc_record_h(const double *m, int32_t stride, double *h)
{
    if (stride == 13) { h[0] = m[10]; h[1] = m[11]; h[2] = m[12]; return; }
    const double *t = m + 10;
    for (int i = 0; i < 3; ++i) { h[i] = 0.0; for (int k = 0; k < 3; ++k) h[i] += t[sym3(i, k, k)]; }
}

/* eps^2 stabiliser.  PAPER.md:107 says only "a small, positive coefficient".  Reading R2-e (UNPINNED):
 * eps2 = eps2_scale * |det(P - theta I)| / (tau theta^4).  Returned here in scaled form
 * eps2_hat = eps2 * tau * theta = eps2_scale * |det(P/theta - I)|. */
static double orc_eps2_hat(const double *Ph /* P/theta, 6 */, double eps2_scale)
{
    double a = Ph[0] - 1.0, b = Ph[1], c = Ph[2], d = Ph[3] - 1.0, e = Ph[4], f = Ph[5] - 1.0;
    double det = a * (d * f - e * e) - b * (b * f - e * c) + c * (b * e - d * c);
    return eps2_scale * fabs(det);
}

/* ------------------------------------------------------------------------------------------------
 * S2+S3 / R2+R3 -- exact cubic-FP closure: assemble and solve the 9x9 moment-matching system.
 * PAPER.md: Eq. 3 (:69) matching condition, Eq. 8 (:102) drift, Eq. 9 (:113) diffusion, Eq. 10 (:121) block
 * form, Table 1 (:130-136) blocks V and W, :124 (right-hand side from Boltzmann relaxation rates), :37/:87
 * (Pr 2/3), Eq. 6 (:83) tau = 2 mu / p, :148 noise sqrt(2 theta/tau).
 * The paper prints only V and W (V rows 5-6 garbled); X^T, Z, Q6, R3 are not printed.  All blocks are
 * therefore DERIVED here from d<psi>/dt = <A_k dpsi/dc_k> + (theta/tau) <Laplacian psi> (R2-d) with Maxwell-
 * molecule rates (R2-f):
 *   psi = c_i c_j   :  c_ik P_kj + c_jk P_ki + gam_i h_j + gam_j h_i = -(2/tau) P_ij + 2 eps2 F_ij
 *   psi = c_i c^2   :  c_ik h_k + 2 c_kl t_kli + gam_i (F - 9 theta^2) + 2 gam_k (F_ki - 3 theta P_ki)
 *                         = -(4/(3 tau)) h_i + eps2 (3 g_i - 3 theta h_i - 2 P_ik h_k)
 * with unknowns y = (c11,c12,c13,c22,c23,c33,gam1,gam2,gam3) (PAPER.md:119 with gamma_1 restored, R2-b) and
 * rows (11,12,13,22,23,33,q1,q2,q3).  The system is assembled from these index formulas by loops (not from a
 * typed-out table) in scaled variables (R3-a): velocity unit sqrt(theta), time unit tau.
 * Solve: Gaussian elimination with partial pivoting (R3-b).  kappa_1 = ||A||_1 ||A^-1||_1 of the scaled
 * matrix from nine extra solves.  Policy for low-count / singular cells: R3-c (UNPINNED).
 * Outputs: coef[9] (double), flag, kappa (nullable).  A_out/b_out (nullable) receive the scaled system.
 * ------------------------------------------------------------------------------------------------ */
static void orc_assemble_scaled(const double *m /* FULL record */, double eps2_scale, double A[9][9], double b[9])
{
    const double *Pm = m + 4, *tm = m + 10, *Fm = m + 20, *gm = m + 26;
    double theta = (Pm[0] + Pm[3] + Pm[5]) / 3.0;
    double s1 = sqrt(theta), s2 = theta, s3 = theta * s1, s4 = theta * theta, s5 = s4 * s1;
    double P[6], t[10], Fij[6], g[3], h[3], F = 0.0;
    for (int k = 0; k < 6; ++k) { P[k] = Pm[k] / s2; Fij[k] = Fm[k] / s4; }
    for (int k = 0; k < 10; ++k) t[k] = tm[k] / s3;
    for (int k = 0; k < 3; ++k) g[k] = gm[k] / s5;
    for (int i = 0; i < 3; ++i) { h[i] = 0.0; for (int k = 0; k < 3; ++k) h[i] += t[sym3(i, k, k)]; F += Fij[sym2(i, i)]; }
    double e2 = orc_eps2_hat(P, eps2_scale);
    memset(A, 0, sizeof(double) * 81);
    /* stress rows (i<=j): c_ik P_kj + c_jk P_ki + gam_i h_j + gam_j h_i = -2 P_ij + 2 e2 F_ij   (theta_hat = tau_hat = 1) */
    for (int i = 0; i < 3; ++i)
        for (int j = i; j < 3; ++j) {
            int r = sym2(i, j);
            for (int k = 0; k < 3; ++k) {
                A[r][sym2(i, k)] += P[sym2(k, j)];
                A[r][sym2(j, k)] += P[sym2(k, i)];
            }
            A[r][6 + i] += h[j];
            A[r][6 + j] += h[i];
            b[r] = -2.0 * P[r] + 2.0 * e2 * Fij[r];
        }
    /* heat-flux rows */
    for (int i = 0; i < 3; ++i) {
        int r = 6 + i;
        for (int k = 0; k < 3; ++k) A[r][sym2(i, k)] += h[k];
        for (int k = 0; k < 3; ++k) for (int l = 0; l < 3; ++l) A[r][sym2(k, l)] += 2.0 * t[sym3(k, l, i)];
        A[r][6 + i] += F - 9.0;
        for (int k = 0; k < 3; ++k) A[r][6 + k] += 2.0 * (Fij[sym2(k, i)] - 3.0 * P[sym2(k, i)]);
        double Ph = 0.0;
        for (int k = 0; k < 3; ++k) Ph += P[sym2(i, k)] * h[k];
        b[r] = -(4.0 / 3.0) * h[i] + e2 * (3.0 * g[i] - 3.0 * h[i] - 2.0 * Ph);
    }
}

/* Gaussian elimination with partial (row) pivoting on a copy; returns the smallest |pivot| met. */
static double orc_ge_solve(const double A0[9][9], const double *b0, double *y)
{
    double A[9][10];
    for (int i = 0; i < 9; ++i) { for (int j = 0; j < 9; ++j) A[i][j] = A0[i][j]; A[i][9] = b0[i]; }
    double minpiv = INFINITY;
    for (int k = 0; k < 9; ++k) {
        int piv = k; double best = fabs(A[k][k]);
        for (int i = k + 1; i < 9; ++i) if (fabs(A[i][k]) > best) { best = fabs(A[i][k]); piv = i; }
        if (piv != k) for (int j = 0; j < 10; ++j) { double s = A[k][j]; A[k][j] = A[piv][j]; A[piv][j] = s; }
        if (!(best >= 0.0)) best = 0.0;               /* NaN */
        if (best < minpiv) minpiv = best;
        if (best == 0.0) { for (int i = 0; i < 9; ++i) y[i] = NAN; return 0.0; }
        for (int i = k + 1; i < 9; ++i) {
            double f = A[i][k] / A[k][k];
            for (int j = k; j < 10; ++j) A[i][j] -= f * A[k][j];
        }
    }
    for (int i = 8; i >= 0; --i) {
        double s = A[i][9];
        for (int j = i + 1; j < 9; ++j) s -= A[i][j] * y[j];
        y[i] = s / A[i][i];
    }
    return minpiv;
}

static void orc_langevin(double tau, double *coef)
{   /* Eq. 4 (:77): A_i = -(1/tau) c_i  <=>  c_ij = -delta_ij/tau, gamma = 0 */
    coef[0] = -1.0 / tau; coef[1] = 0; coef[2] = 0; coef[3] = -1.0 / tau; coef[4] = 0; coef[5] = -1.0 / tau;
    coef[6] = 0; coef[7] = 0; coef[8] = 0;
}

void orc_closure_exact_cell(const double *m, double tau, double eps2_scale, int32_t min_count,
                            double *coef, uint32_t *flag, double *kappa, double *A_out, double *b_out)
{
    *flag = 0;
    if (kappa) *kappa = 0.0;
    double n = m[0];
    if (n <= 0.0) { for (int k = 0; k < 9; ++k) coef[k] = 0.0; *flag = ORC_FLAG_EMPTY; return; }
    double theta = (m[4] + m[7] + m[9]) / 3.0;
    if (n < (double)min_count) { orc_langevin(tau, coef); *flag = ORC_FLAG_LOWCOUNT; return; }
    if (!(theta > 0.0) || !isfinite(theta)) { orc_langevin(tau, coef); *flag = ORC_FLAG_SINGULAR; return; }
    double A[9][9], b[9], y[9];
    orc_assemble_scaled(m, eps2_scale, A, b);
    if (A_out) memcpy(A_out, A, sizeof(double) * 81);
    if (b_out) memcpy(b_out, b, sizeof(double) * 9);
    double minpiv = orc_ge_solve(A, b, y);
    int finite = 1;
    for (int k = 0; k < 9; ++k) if (!isfinite(y[k])) finite = 0;
    if (!(minpiv >= 1e-14) || !finite) { orc_langevin(tau, coef); *flag = ORC_FLAG_SINGULAR; return; }
    /* kappa_1 of the scaled matrix: ||A||_1 (max column sum) times ||A^-1||_1 from nine unit-vector solves */
    double nA = 0.0, nAi = 0.0;
    for (int j = 0; j < 9; ++j) { double s = 0; for (int i = 0; i < 9; ++i) s += fabs(A[i][j]); if (s > nA) nA = s; }
    for (int j = 0; j < 9; ++j) {
        double e[9] = {0}, z[9]; e[j] = 1.0;
        orc_ge_solve(A, e, z);
        double s = 0; for (int i = 0; i < 9; ++i) s += fabs(z[i]);
        if (s > nAi) nAi = s;
    }
    double kap = nA * nAi;
    if (kappa) *kappa = kap;
    if (!(kap < 1e8)) *flag |= ORC_FLAG_ILLCOND;
    /* un-scale: c = c_hat / tau, gamma = gamma_hat / (tau sqrt(theta)) */
    for (int k = 0; k < 6; ++k) coef[k] = y[k] / tau;
    for (int k = 6; k < 9; ++k) coef[k] = y[k] / (tau * sqrt(theta));
}

/* Batched form.  tau_cell nullable (then tau_scalar is used); kappa nullable. */
void orc_closure_exact(int32_t ncell, const double *mom_full, const float *tau_cell, double tau_scalar,
                       double eps2_scale, int32_t min_count, double *coef, uint32_t *flags, double *kappa)
{
#pragma omp parallel for schedule(dynamic, 64)
    for (int32_t c = 0; c < ncell; ++c) {
        double tau = tau_cell ? (double)tau_cell[c] : tau_scalar;
        orc_closure_exact_cell(mom_full + (size_t)c * 29, tau, eps2_scale, min_count, coef + (size_t)c * 9,
                               flags + c, kappa ? kappa + c : NULL, NULL, NULL);
    }
}

/* ------------------------------------------------------------------------------------------------
 * NEXT-2: sampling outputs.
 * Per-cell nonequilibrium diagnostics from the FULL record (R_ij = <c_i c_j c_k c_k>,
 * Delta_4 = <(c_k c_k)^2> - 15 theta^2, theta = <c_k c_k>/3; Eq. 19-23 :632-657: Theta_ij = <c_i c_j>,
 * D_G = -1/2 log det(Theta/theta), ds_eq = 3/2 log(theta/theta_inf) - log(rho/rho_inf),
 * ds_kin,G = ds_eq - (D_G - D_G,inf), D_q = |q_hat|^2 / 5 with q_hat = <c |c|^2> / (2 theta^(3/2))).
 * "norm" = divided by the local Maxwellian scale (reading R10: the paper only says
 * "nondimensionalization by the corresponding local Maxwellian scales"): Delta_4 / (15 theta^2),
 * R_ij / (5 theta^2) (a Maxwellian has <c_i c_j c^2> = 5 theta^2 delta_ij), sigma_norm = |P - theta I|_F / theta,
 * q_norm = |q_hat|, m3_norm = |t|_F / theta^(3/2) (all 27 index triples).  DM6 = <(c^2)^3> needs a sixth-order
 * accumulator that the FULL record does not carry and is not produced.
 * diag record (16): theta, Delta_4, Delta_4/(15 theta^2), D_G, D_q, ds_eq, ds_kin,G, sigma_norm, q_norm, m3_norm,
 *                   R_11, R_12, R_13, R_22, R_23, R_33 (each / (5 theta^2)).
 * Empty cell or theta <= 0: zeros.  Singular covariance: D_G = +inf, ds_kin,G = -inf; "singular" is N < 4 (the
 * covariance of N points has rank <= N - 1, its determinant is zero up to rounding, and the sign of that rounding
 * must not decide the result) or det(Theta/theta) <= 0 (a degenerate cloud).  rho/rho_inf is N / n_inf (uniform particle weight).
 * ------------------------------------------------------------------------------------------------ */
void orc_cell_diagnostics(int32_t ncell, const double *mom_full, double theta_inf, double n_inf, double dg_inf,
                          double *diag)
{
    static const double mult3[10] = {1, 3, 3, 3, 6, 3, 1, 3, 3, 1};       /* 111,112,113,122,123,133,222,223,233,333 */
    for (int32_t cell = 0; cell < ncell; ++cell) {
        const double *m = mom_full + (size_t)cell * 29;
        double *d = diag + (size_t)cell * 16;
        for (int k = 0; k < 16; ++k) d[k] = 0.0;
        const double N = m[0];
        const double *P = m + 4, *t = m + 10, *F = m + 20;
        const double theta = (P[0] + P[3] + P[5]) / 3.0;
        if (!(N > 0.0) || !(theta > 0.0)) continue;
        const double c4 = F[0] + F[3] + F[5];                              /* <c^4> = F_kk */
        d[0] = theta;
        d[1] = c4 - 15.0 * theta * theta;
        d[2] = d[1] / (15.0 * theta * theta);
        const double a = P[0] / theta, b = P[1] / theta, c = P[2] / theta, e = P[3] / theta, f = P[4] / theta,
                     g = P[5] / theta;                                     /* Theta/theta = [[a,b,c],[b,e,f],[c,f,g]] */
        const double det = a * (e * g - f * f) - b * (b * g - f * c) + c * (b * f - e * c);
        d[3] = (N >= 4.0 && det > 0.0) ? -0.5 * log(det) : INFINITY;
        double h[3];
        orc_record_h(m, 29, h);
        const double qn = sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]) / (2.0 * theta * sqrt(theta));
        d[4] = qn * qn / 5.0;
        d[5] = 1.5 * log(theta / theta_inf) - log(N / n_inf);
        d[6] = d[5] - (d[3] - dg_inf);
        const double sxx = P[0] - theta, syy = P[3] - theta, szz = P[5] - theta;
        d[7] = sqrt(sxx * sxx + syy * syy + szz * szz + 2.0 * (P[1] * P[1] + P[2] * P[2] + P[4] * P[4])) / theta;
        d[8] = qn;
        double t2 = 0.0;
        for (int k = 0; k < 10; ++k) t2 += mult3[k] * t[k] * t[k];
        d[9] = sqrt(t2) / (theta * sqrt(theta));
        for (int k = 0; k < 6; ++k) d[10 + k] = F[k] / (5.0 * theta * theta);
    }
}

/* DM6 = <(c_k c_k)^3>, the sixth central moment of PAPER.md:415, per cell from the cell-sorted particles (the FULL
 * record stops at fifth order).  dm6[cell] = (1/N) sum (|v - U|^2)^3 with U the cell mean (recomputed here); empty
 * cell: 0.  A Maxwellian has <c^6> = 105 theta^3, which is the "local Maxwellian scale" of DM6_norm (reading R10). */
void orc_cell_dm6(const float *vx, const float *vy, const float *vz, const int32_t *cell_start, int32_t ncell, double *dm6)
{
    for (int32_t cell = 0; cell < ncell; ++cell) {
        int64_t s = cell_start[cell], e = cell_start[cell + 1], n = e - s;
        dm6[cell] = 0.0;
        if (n <= 0) continue;
        double U[3] = {0, 0, 0};
        for (int64_t p = s; p < e; ++p) { U[0] += vx[p]; U[1] += vy[p]; U[2] += vz[p]; }
        for (int i = 0; i < 3; ++i) U[i] /= (double)n;
        double acc = 0.0;
        for (int64_t p = s; p < e; ++p) {
            double c0 = (double)vx[p] - U[0], c1 = (double)vy[p] - U[1], c2 = (double)vz[p] - U[2];
            double r2 = c0 * c0 + c1 * c1 + c2 * c2;
            acc += r2 * r2 * r2;
        }
        dm6[cell] = acc / (double)n;
    }
}

/* Running time average of sampled grid fields (PAPER.md:217-219 average_results): after the call avg holds the
 * mean of the k + 1 samples seen so far, avg <- avg + (x - avg) / (k + 1). */
void orc_average_results(int64_t n, const double *x, int64_t k, double *avg)
{
    for (int64_t i = 0; i < n; ++i) avg[i] = avg[i] + (x[i] - avg[i]) / (double)(k + 1);
}

/* ------------------------------------------------------------------------------------------------
 * S4 / R4 -- MLP surrogate.  PAPER.md:233 (16 features), :234 (9 targets), :242 (W, b, mu, sigma exported),
 * :264 (predict_coeffs), :309 (16-256-256-256-256-9, ReLU, 204,041 parameters), :327 (StandardScaler on
 * inputs and outputs), :568 (under-relaxation w).
 * Features from the moment record in fp64, cast to fp32 (the network's input precision); then
 * z = (x - x_mean)/x_scale, hidden layers z <- act(W z + b), head linear, y = yhat*y_scale + y_mean, all
 * accumulated in fp64 from the fp32 weights.  W is row-major [out][in].  act 0 = SiLU x/(1+e^-x), 1 = ReLU.
 * feature_set 0 (BASELINE.json, 13): n, U1,U2,U3, T, pi11,pi12,pi13,pi22,pi23, q1,q2,q3 with n = N*n_scale,
 *   T = theta/theta_ref, pi_ij = n (P_ij - theta delta_ij), q_i = n h_i / 2  (R4; pi33 dropped as redundant).
 * feature_set 1 (paper's 16, definitions UNPINNED R4): rho=n, T, U(3), Pi_ij = n P_ij (6), q(3),
 *   DM2 = 3 theta, nu = 1/tau.
 * relax_w: coef <- w*new + (1-w)*old; w = 1 overwrites (old is not read); a cell whose old coefficients
 * are all exactly zero (EMPTY at the previous step, zero-initialised first step) has no history and is not blended (R12).
 * Flags: EMPTY -> zeros; N < min_count or theta <= 0 -> Langevin, LOWCOUNT/SINGULAR; non-finite output ->
 * Langevin + NONFINITE.
 * ------------------------------------------------------------------------------------------------ */
int32_t orc_mlp_features(const double *m, int32_t stride, int32_t feature_set, double n_scale, double theta_ref,
                         double tau, float *x)
{
    double h[3];
    orc_record_h(m, stride, h);
    double n = m[0] * n_scale;
    double theta = (m[4] + m[7] + m[9]) / 3.0;
    if (feature_set == 0) {
        x[0] = (float)n; x[1] = (float)m[1]; x[2] = (float)m[2]; x[3] = (float)m[3];
        x[4] = (float)(theta / theta_ref);
        x[5] = (float)(n * (m[4] - theta)); x[6] = (float)(n * m[5]); x[7] = (float)(n * m[6]);
        x[8] = (float)(n * (m[7] - theta)); x[9] = (float)(n * m[8]);
        for (int i = 0; i < 3; ++i) x[10 + i] = (float)(0.5 * n * h[i]);
        return 13;
    }
    x[0] = (float)n; x[1] = (float)(theta / theta_ref);
    x[2] = (float)m[1]; x[3] = (float)m[2]; x[4] = (float)m[3];
    for (int k = 0; k < 6; ++k) x[5 + k] = (float)(n * m[4 + k]);
    for (int i = 0; i < 3; ++i) x[11 + i] = (float)(0.5 * n * h[i]);
    x[14] = (float)(3.0 * theta);
    x[15] = (float)(1.0 / tau);
    return 16;
}

void orc_mlp_forward(int32_t n_layers, const int32_t *dims, const float *const *W, const float *const *b,
                     const float *x_mean, const float *x_scale, const float *y_mean, const float *y_scale,
                     int32_t act, const float *x, double *y)
{
    double z[1024], zn[1024];
    int nin = dims[0];
    for (int i = 0; i < nin; ++i) z[i] = ((double)x[i] - (double)x_mean[i]) / (double)x_scale[i];
    for (int l = 0; l < n_layers; ++l) {
        int ni = dims[l], no = dims[l + 1];
        for (int o = 0; o < no; ++o) {
            double s = (double)b[l][o];
            for (int i = 0; i < ni; ++i) s += (double)W[l][(size_t)o * ni + i] * z[i];
            if (l < n_layers - 1) s = (act == 0) ? s / (1.0 + exp(-s)) : (s > 0.0 ? s : 0.0);
            zn[o] = s;
        }
        for (int o = 0; o < no; ++o) z[o] = zn[o];
    }
    int nout = dims[n_layers];
    for (int o = 0; o < nout; ++o) y[o] = z[o] * (double)y_scale[o] + (double)y_mean[o];
}

void orc_closure_mlp(int32_t ncell, const double *mom, int32_t stride, const float *tau_cell, double tau_scalar,
                     int32_t n_layers, const int32_t *dims, const float *const *W, const float *const *b,
                     const float *x_mean, const float *x_scale, const float *y_mean, const float *y_scale,
                     int32_t act, int32_t feature_set, double n_scale, double theta_ref, int32_t min_count,
                     double relax_w, const double *coef_old, double *coef, uint32_t *flags)
{
#pragma omp parallel for schedule(dynamic, 64)
    for (int32_t c = 0; c < ncell; ++c) {
        const double *m = mom + (size_t)c * stride;
        double *out = coef + (size_t)c * 9;
        double tau = tau_cell ? (double)tau_cell[c] : tau_scalar;
        double y[9];
        uint32_t flag = 0;
        double theta = (m[4] + m[7] + m[9]) / 3.0;
        if (m[0] <= 0.0) { for (int k = 0; k < 9; ++k) out[k] = 0.0; flags[c] = ORC_FLAG_EMPTY; continue; }
        if (m[0] < (double)min_count) { orc_langevin(tau, y); flag = ORC_FLAG_LOWCOUNT; }
        else if (!(theta > 0.0) || !isfinite(theta)) { orc_langevin(tau, y); flag = ORC_FLAG_SINGULAR; }
        else {
            float x[16];
            orc_mlp_features(m, stride, feature_set, n_scale, theta_ref, tau, x);
            orc_mlp_forward(n_layers, dims, W, b, x_mean, x_scale, y_mean, y_scale, act, x, y);
            int finite = 1;
            for (int k = 0; k < 9; ++k) if (!isfinite(y[k])) finite = 0;
            if (!finite) { orc_langevin(tau, y); flag = ORC_FLAG_NONFINITE; }
        }
        /* reading R12: a cell without history -- all nine old coefficients exactly zero: it was EMPTY at the previous
         * step, or this is the first step on a zero-initialised array -- takes the new values unblended */
        int history = 0;
        if (relax_w != 1.0) for (int k = 0; k < 9; ++k) if (coef_old[(size_t)c * 9 + k] != 0.0) history = 1;
        for (int k = 0; k < 9; ++k)
            out[k] = history ? relax_w * y[k] + (1.0 - relax_w) * coef_old[(size_t)c * 9 + k] : y[k];
        flags[c] = flag;
    }
}

/* ------------------------------------------------------------------------------------------------
 * S6 / R6 -- counter-based normals.  PAPER.md:163 says only "standard normal random variate"; the north star
 * fixes Philox.  Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11 -- the public algorithm): multipliers
 * 0xD2511F53, 0xCD9E8D57; Weyl key increments 0x9E3779B9, 0xBB67AE85; ten rounds, key bumped between rounds.
 * counter = (pid, step_lo, step_hi, stream), key = (seed_lo, seed_hi).
 * word -> uniform: u = ((w >> 9) + 0.5) * 2^-23, exact in fp32, in (0,1).
 * Box-Muller: xi1 = sqrt(-2 ln u0) cos(2 pi u1), xi2 = sqrt(-2 ln u0) sin(2 pi u1), xi3 = sqrt(-2 ln u2) cos(2 pi u3),
 * evaluated in fp64 from the same u.
 * ------------------------------------------------------------------------------------------------ */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0, hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

static double orc_uniform(uint32_t w) { return ((double)(w >> 9) + 0.5) * (1.0 / 8388608.0); }

void orc_uniforms(uint32_t pid, uint64_t step, uint32_t stream, uint64_t seed, double u[4])
{
    uint32_t ctr[4] = {pid, (uint32_t)step, (uint32_t)(step >> 32), stream};
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)}, w[4];
    orc_philox4x32_10(ctr, key, w);
    for (int i = 0; i < 4; ++i) u[i] = orc_uniform(w[i]);
}

void orc_normals(uint32_t pid, uint64_t step, uint32_t stream, uint64_t seed, double xi[3])
{
    double u[4];
    orc_uniforms(pid, step, stream, seed, u);
    double r0 = sqrt(-2.0 * log(u[0])), r1 = sqrt(-2.0 * log(u[2]));
    xi[0] = r0 * cos(2.0 * ORC_PI * u[1]);
    xi[1] = r0 * sin(2.0 * ORC_PI * u[1]);
    xi[2] = r1 * cos(2.0 * ORC_PI * u[3]);
}

/* ------------------------------------------------------------------------------------------------
 * S5 / R5 -- FP velocity update.  PAPER.md: Eq. 13 (:156), definitions (:161-165), Eq. 14 (:171), :174,
 * Eq. 15 (:178), :181 (plain mean), :463 (momentum recentred, energy controlled by the alpha rescaling).
 * Per cell with N >= 2 and theta > 0 (otherwise velocities untouched, SKIPPED):
 *  1. U, theta = P_kk/3, h from the record of the same pre-update particles; a = dt/tau, E1 = e^-a, E2 = e^-2a;
 *     eps2 = eps2_scale |det(P - theta I)| / (tau theta^4)  (R2-e).
 *  2. c = v - U (":161 M'_i = M_i U_i": the minus sign is lost in the extraction);
 *     N_i = (C_ij + delta_ij/tau) c_j + gam_i (c^2 - 3 theta) - eps2 (c_i c^2 - h_i)          (Eq. 14; 2q_i/rho = h_i)
 *  3. alpha^2 = 1 + tau/(3 theta) [ tau (1-E1)^2 <N.N> + 2 (E1 - E2) <c.N> ]                    (Eq. 15)
 *     non-finite or < 1e-6 -> alpha = 1, flag ALPHA.
 *  4. xi from Philox(pid, step, stream 0);  c* = (1/alpha)[c E1 + (1-E1) tau N + sqrt(theta (1-E2)) xi]   (Eq. 13)
 *  5. conserve_mode 0: c_new = c*.  conserve_mode 1 (R5.5): m = <c*>, c0 = c* - m, e = <|c0|^2>,
 *     c_new = c0 sqrt(3 theta / e)  (exact momentum and energy conservation per cell; if e <= 0, no rescale).
 *  6. v <- U + c_new, rounded to fp32.
 * coef is the fp32 array the closure wrote (the GPU consumes the same values).
 * ------------------------------------------------------------------------------------------------ */
void orc_velocity_update(int32_t ncell, const int32_t *cell_start, float *vx, float *vy, float *vz,
                         const uint32_t *pid, const double *mom, int32_t stride, const float *coef,
                         const float *tau_cell, double tau_scalar, double dt, double eps2_scale,
                         int32_t conserve_mode, uint64_t seed, uint64_t step, uint32_t *flags)
{
#pragma omp parallel for schedule(dynamic, 64)
    for (int32_t cell = 0; cell < ncell; ++cell) {
        int64_t s = cell_start[cell], e = cell_start[cell + 1], n = e - s;
        const double *m = mom + (size_t)cell * stride;
        double tau = tau_cell ? (double)tau_cell[cell] : tau_scalar;
        double theta = (m[4] + m[7] + m[9]) / 3.0;
        if (n < 2 || !(theta > 0.0) || !isfinite(theta)) { if (n > 0) flags[cell] |= ORC_FLAG_SKIPPED; continue; }
        double U[3] = {m[1], m[2], m[3]}, h[3];
        orc_record_h(m, stride, h);
        double Ph[6];
        for (int k = 0; k < 6; ++k) Ph[k] = m[4 + k] / theta;
        double eps2 = orc_eps2_hat(Ph, eps2_scale) / (tau * theta);
        const float *cf = coef + (size_t)cell * 9;
        double C[3][3] = {{cf[0], cf[1], cf[2]}, {cf[1], cf[3], cf[4]}, {cf[2], cf[4], cf[5]}};
        double gam[3] = {cf[6], cf[7], cf[8]};
        double a = dt / tau, E1 = exp(-a), E2 = exp(-2.0 * a);
        double *Nv = (double *)malloc(sizeof(double) * 3 * (size_t)n);
        double *cs = (double *)malloc(sizeof(double) * 3 * (size_t)n);
        double sNN = 0.0, scN = 0.0;
        for (int64_t p = 0; p < n; ++p) {
            double c[3] = {(double)vx[s + p] - U[0], (double)vy[s + p] - U[1], (double)vz[s + p] - U[2]};
            double c2 = c[0] * c[0] + c[1] * c[1] + c[2] * c[2];
            for (int i = 0; i < 3; ++i) {
                double Ni = 0.0;
                for (int j = 0; j < 3; ++j) Ni += (C[i][j] + (i == j ? 1.0 / tau : 0.0)) * c[j];
                Ni += gam[i] * (c2 - 3.0 * theta) - eps2 * (c[i] * c2 - h[i]);
                Nv[3 * p + i] = Ni;
                sNN += Ni * Ni; scN += c[i] * Ni;
            }
        }
        sNN /= (double)n; scN /= (double)n;
        double alpha2 = 1.0 + tau / (3.0 * theta) * (tau * (1.0 - E1) * (1.0 - E1) * sNN + 2.0 * (E1 - E2) * scN);
        double alpha = 1.0;
        if (!isfinite(alpha2) || alpha2 < 1e-6) flags[cell] |= ORC_FLAG_ALPHA; else alpha = sqrt(alpha2);
        double sig = sqrt(theta * (1.0 - E2));
        double mean[3] = {0, 0, 0};
        for (int64_t p = 0; p < n; ++p) {
            double xi[3];
            orc_normals(pid[s + p], step, 0u, seed, xi);
            double c[3] = {(double)vx[s + p] - U[0], (double)vy[s + p] - U[1], (double)vz[s + p] - U[2]};
            for (int i = 0; i < 3; ++i) {
                cs[3 * p + i] = (c[i] * E1 + (1.0 - E1) * tau * Nv[3 * p + i] + sig * xi[i]) / alpha;
                mean[i] += cs[3 * p + i];
            }
        }
        if (conserve_mode == 1) {
            for (int i = 0; i < 3; ++i) mean[i] /= (double)n;
            double en = 0.0;
            for (int64_t p = 0; p < n; ++p) for (int i = 0; i < 3; ++i) { cs[3 * p + i] -= mean[i]; en += cs[3 * p + i] * cs[3 * p + i]; }
            en /= (double)n;
            double sc = (en > 0.0 && isfinite(en)) ? sqrt(3.0 * theta / en) : 1.0;
            for (int64_t p = 0; p < 3 * n; ++p) cs[p] *= sc;
        }
        for (int64_t p = 0; p < n; ++p) {
            vx[s + p] = (float)(U[0] + cs[3 * p + 0]);
            vy[s + p] = (float)(U[1] + cs[3 * p + 1]);
            vz[s + p] = (float)(U[2] + cs[3 * p + 2]);
        }
        free(Nv); free(cs);
    }
}

/* ------------------------------------------------------------------------------------------------
 * S7 / R7 -- streaming and diffuse isothermal walls.  PAPER.md: Eq. 16 (:187) X <- X + M dt, :213-214
 * (Move_Particles_2D, Apply_Boundary_Cavity), :380 (cavity), :278-282 (Couette plates), :674 ("diffuse
 * reflection from an isothermal wall").  The paper gives no re-emission details; reading R7 (UNPINNED against
 * the paper's runs; pinned against the half-range Maxwellian):
 *   x <- fmaf(vx, dt, x), y <- fmaf(vy, dt, y) in fp32 (positions decide the cell index, so the fp32 sequence
 *   is part of the definition).  Then x-pair, y-pair, embedded body, in this order.
 *   Beyond a diffuse wall at xw: x <- xw + (xw - x) in fp32, clamped into [xmin, pred(xmax)] if still outside;
 *   velocity redrawn from one Philox call (stream 1 = x-pair, 2 = y-pair, 4 = body): normal component
 *   sqrt(-2 theta_w ln u0) into the gas, tangentials U_w,t + sqrt(theta_w) * (Box-Muller pair from u1, u2).
 *   Periodic: x <- x -/+ (xmax - xmin).  kind 0 (none): nothing.
 *   Body (cylinder, centre (cx,cy), radius R): r2 = fmaf(dy,dy,dx*dx) < R*R -> moved radially to
 *   R*1.000001f: s = (R*1.000001f)/sqrtf(r2), x = fmaf(dx, s, cx) (fp32); velocity redrawn about the
 *   outward normal n = (dx,dy)/r, tangent (-n_y, n_x), and z.
 *   kind 3 (freestream reservoir, reading R11; SURVEY S7 "outer faces are a constant-Np reservoir: a particle leaving is
 *   re-inserted on the inflow face with a flux-weighted freestream velocity", PAPER.md:545 Mach-10 argon freestream):
 *   the freestream (theta_inf; U_inf with U_inf,x > 0) is wall[0]'s (theta_w; ux, uy, uz) and the inflow face is xmin.
 *   A particle that leaves through a kind-3 face is re-inserted at xmin:
 *     v_x from the flux-weighted drifting half-Maxwellian f(v) ~ v exp(-(v - U)^2 / (2 theta)), v > 0, by acceptance-
 *       rejection: mu = (U + sqrt(U^2 + 4 theta)) / 2 (the mode of f), candidate v = mu + sqrt(theta) z with
 *       z = sqrt(-2 ln u0) cos(2 pi u1), accepted iff v > 0 and (v / mu) exp(1 - v / mu) >= u2 (f / proposal, scaled to 1 at
 *       the mode); attempt a = 0..7 uses the Philox call with stream 16 + a; if all eight are rejected, v = mu;
 *     v_y = U_y + t1, v_z = U_z + t2 with (t1, t2) = sqrt(theta) sqrt(-2 ln u0) (cos, sin)(2 pi u1) from the call with stream 32;
 *     position, in fp32 (it decides the cell): x = xmin + u3 * fl(U_x * dt) (the particle entered at a uniformly distributed
 *       moment of the step), y = fmaf(u2, Ly, ymin) (uniform along the face; 1D: y unchanged), clamped into the domain;
 *     no further wall of this step applies to it (the body test still does).
 * wall[k] = {kind, theta_w, ux, uy, uz} for k = xmin, xmax, ymin, ymax, given as 5 doubles each (kind as a number).
 * ------------------------------------------------------------------------------------------------ */
static void orc_wall_draw(uint32_t pid, uint64_t step, uint32_t stream, uint64_t seed, double theta_w,
                          double *vn, double *t1, double *t2)
{
    double u[4];
    orc_uniforms(pid, step, stream, seed, u);
    *vn = sqrt(-2.0 * theta_w * log(u[0]));
    double r = sqrt(-2.0 * log(u[1])), st = sqrt(theta_w);
    *t1 = st * r * cos(2.0 * ORC_PI * u[2]);
    *t2 = st * r * sin(2.0 * ORC_PI * u[2]);
}

static void orc_reinsert(uint32_t pid, uint64_t step, uint64_t seed, const double *w0, float xmin, float xmax, float ymin,
                         float ymax, float Ly, float pen, int two_d, float *xp, float *yp, double v[3])
{
    double th = w0[1], U = w0[2], sg = sqrt(th), mu = 0.5 * (U + sqrt(U * U + 4.0 * th)), vn = mu, u[4];
    for (uint32_t a = 0; a < 8; ++a) {
        orc_uniforms(pid, step, 16u + a, seed, u);
        double c = mu + sg * sqrt(-2.0 * log(u[0])) * cos(2.0 * ORC_PI * u[1]);
        if (c > 0.0 && (c / mu) * exp(1.0 - c / mu) >= u[2]) { vn = c; break; }
    }
    orc_uniforms(pid, step, 32u, seed, u);
    double r = sg * sqrt(-2.0 * log(u[0]));
    v[0] = vn; v[1] = w0[3] + r * cos(2.0 * ORC_PI * u[1]); v[2] = w0[4] + r * sin(2.0 * ORC_PI * u[1]);
    float u2f = (float)u[2], u3f = (float)u[3];          /* (k + 1/2) 2^-23: exact in fp32 */
    float xn = xmin + u3f * pen;
    if (xn < xmin) xn = xmin;
    if (xn >= xmax) xn = nextafterf(xmax, -INFINITY);
    *xp = xn;
    if (two_d) {
        float yn = fmaf(u2f, Ly, ymin);
        if (yn < ymin) yn = ymin;
        if (yn >= ymax) yn = nextafterf(ymax, -INFINITY);
        *yp = yn;
    }
}

void orc_stream_walls(int64_t np, float *x, float *y, float *vx, float *vy, float *vz, const uint32_t *pid,
                      int32_t nx, int32_t ny, float x0, float y0, float dx, float dy, float dt,
                      const double *wall /* 4 x 5 */, int32_t body_kind, float bcx, float bcy, float bR,
                      double body_theta_w, uint64_t seed, uint64_t step)
{
    float xmin = x0, xmax = x0 + (float)nx * dx, ymin = y0, ymax = y0 + (float)ny * dy;
    float Lx = xmax - xmin, Ly = ymax - ymin;
    float pen = (float)wall[2] * dt;                       /* fp32: fl(U_inf,x) * dt, one rounding */
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < np; ++p) {
        float xp = fmaf(vx[p], dt, x[p]), yp = fmaf(vy[p], dt, y[p]);
        double v[3] = {vx[p], vy[p], vz[p]};
        int redrawn = 0, reinserted = 0;
        /* x pair */
        {
            int side = (xp < xmin) ? 0 : ((xp >= xmax) ? 1 : -1);
            if (side >= 0) {
                const double *w = wall + 5 * side;
                int kind = (int)w[0];
                float xw = side ? xmax : xmin;
                if (kind == 1) {
                    float t = xw - xp; xp = xw + t;
                    if (xp < xmin) xp = xmin;
                    if (xp >= xmax) xp = nextafterf(xmax, -INFINITY);
                    double vn, t1, t2;
                    orc_wall_draw(pid[p], step, 1u, seed, w[1], &vn, &t1, &t2);
                    v[0] = side ? -vn : vn; v[1] = w[3] + t1; v[2] = w[4] + t2; redrawn = 1;
                } else if (kind == 2) {
                    xp = side ? xp - Lx : xp + Lx;
                    if (xp < xmin) xp = xmin;
                    if (xp >= xmax) xp = nextafterf(xmax, -INFINITY);
                } else if (kind == 3) {
                    orc_reinsert(pid[p], step, seed, wall, xmin, xmax, ymin, ymax, Ly, pen, ny > 1, &xp, &yp, v);
                    redrawn = 1; reinserted = 1;
                }
            }
        }
        /* y pair */
        if (ny > 1 && !reinserted) {
            int side = (yp < ymin) ? 0 : ((yp >= ymax) ? 1 : -1);
            if (side >= 0) {
                const double *w = wall + 5 * (2 + side);
                int kind = (int)w[0];
                float yw = side ? ymax : ymin;
                if (kind == 1) {
                    float t = yw - yp; yp = yw + t;
                    if (yp < ymin) yp = ymin;
                    if (yp >= ymax) yp = nextafterf(ymax, -INFINITY);
                    double vn, t1, t2;
                    orc_wall_draw(pid[p], step, 2u, seed, w[1], &vn, &t1, &t2);
                    v[1] = side ? -vn : vn; v[0] = w[2] + t1; v[2] = w[4] + t2; redrawn = 1;
                } else if (kind == 2) {
                    yp = side ? yp - Ly : yp + Ly;
                    if (yp < ymin) yp = ymin;
                    if (yp >= ymax) yp = nextafterf(ymax, -INFINITY);
                } else if (kind == 3) {
                    orc_reinsert(pid[p], step, seed, wall, xmin, xmax, ymin, ymax, Ly, pen, 1, &xp, &yp, v);
                    redrawn = 1;
                }
            }
        }
        /* embedded body */
        if (body_kind == 1) {
            float ddx = xp - bcx, ddy = yp - bcy;
            float r2 = fmaf(ddy, ddy, ddx * ddx);
            if (r2 < bR * bR) {
                float r = sqrtf(r2);
                double nxn, nyn;
                if (r > 0.0f) {
                    float sc = (bR * 1.000001f) / r;
                    nxn = (double)ddx / (double)r; nyn = (double)ddy / (double)r;
                    xp = fmaf(ddx, sc, bcx); yp = fmaf(ddy, sc, bcy);
                } else { nxn = 1.0; nyn = 0.0; xp = bcx + bR * 1.000001f; }
                double vn, t1, t2;
                orc_wall_draw(pid[p], step, 4u, seed, body_theta_w, &vn, &t1, &t2);
                v[0] = vn * nxn - t1 * nyn; v[1] = vn * nyn + t1 * nxn; v[2] = t2; redrawn = 1;
            }
        }
        x[p] = xp; y[p] = yp;
        if (redrawn) { vx[p] = (float)v[0]; vy[p] = (float)v[1]; vz[p] = (float)v[2]; }
    }
}

/* Gather helper for the loop: out[k] = in[perm[k]] (4-byte items). */
void orc_permute_u32(int64_t np, const uint32_t *perm, const uint32_t *in, uint32_t *out)
{
    for (int64_t k = 0; k < np; ++k) out[k] = in[perm[k]];
}

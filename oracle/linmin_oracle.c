/*
 * linmin_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU oracle for the LinMin hot path: per-pixel fully constrained linear
 * unmixing.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call it.  It shares no code with the CUDA path (paper_1402_2518_b200/csrc) and does
 * not use its algorithm: the CUDA path runs an interior-point iteration on the normal equations;
 * this file computes the DEFINITION of the result.
 *
 * What is computed (citations are PAPER.md line + section/equation):
 *   PAPER.md:48-50 (sec. 2.1, eq. 1)  X = A.S + E.  Here (notation of BASELINE.json): a pixel's
 *       spectrum y (L channels), library A (L x R, column r = endmember r), coefficients a (R).
 *   PAPER.md:54 (eq. 2)   F(a) = sum_l ( y_l - (A a)_l )^2, separable per pixel.
 *   PAPER.md:63 (eq. 3)   a_r >= 0.
 *   PAPER.md:68 (eq. 4)   sum_r a_r = 1.
 *   PAPER.md:73 (sec. 2.2) IPLS converges to the minimiser because F is convex; the result of the
 *       method is therefore the minimiser a* of (2) under (3)-(4), which is what this file returns.
 *   PAPER.md:88 (sec. 2.3) "An estimation of the error on the mixing coefficient A is directly
 *       provided by the Hessian": reading R3 of DESIGN.md -- first-order propagation of the
 *       per-channel noise std through the solution map on the optimal support.
 *   PAPER.md:143, 246, 252  "RMS": sqrt(mean_l r_l^2), r = y - A a*  (reading R8).
 *
 * Algorithm (exact in finitely many steps; textbook primal active-set for a convex QP whose
 * equality-constrained sub-problems are solved IN DATA SPACE by Householder QR -- no normal
 * equations, so the squared condition number never appears):
 *   1. widen the fp32 inputs to fp64.
 *   2. start at the best vertex j = argmin_i ||y - A_i||^2, F = {j}, a = e_j.
 *   3. solve min ||y - A_F a_F|| s.t. 1'a_F = 1:  a_F = a0 + Z c, a0 = 1/k, Z an orthonormal basis
 *      of {z : 1'z = 0}, c = argmin ||(y - A_F a0) - (A_F Z) c|| by column-pivoted Householder QR.
 *   4. all a_F > 0: accept; gradient g = A'(A a - y); nu = -g_F'a_F; multipliers
 *      lambda_i = g_i + nu (i not in F).  min lambda >= -(1e-12 ||g||_inf + 1e-13 s): optimal, where
 *      s = max_i sum_l |A_li||y_l| bounds the rounding noise of g itself (without it a noiseless
 *      pixel, g = 0 exactly in theory, would chase fp64 rounding).  Else add argmin.
 *   5. otherwise step from the current point towards the sub-problem solution until the first
 *      coefficient reaches zero, drop it, go to 3.
 *
 * Options added for the NEXT rows of SURVEY.md 8(f) (linmin_oracle_solve_ex; linmin_oracle_solve is the sum-to-one,
 * unweighted case and its arithmetic is unchanged):
 *   constraint (the sto / slo / pos options of IPLS)
 *     sto  eq. 3 + eq. 4, as above.
 *     slo  "sum lower than one": a >= 0, sum a <= 1.  With the slack s = 1 - sum a >= 0 this IS the sto problem on
 *          the library [A | 0] (a zero endmember carries the slack): solved as such, the slack column dropped from
 *          the outputs.
 *     pos  positivity only (eq. 2 under eq. 3; NNLS, PAPER.md:71 cites Lawson-Hanson): the same primal active-set
 *          loop without the equality constraint -- start at a = 0, sub-problems min ||y - A_F a_F|| by Householder
 *          QR of A_F, multipliers lambda_i = g_i, uncertainties through J = A_F^+ .
 *   weighting (eq. 5-6): one noise covariance C (L x L) for the whole image.  Eq. 6 is eq. 2 on
 *          X' = X.L, S' = S.L with C^-1 = L.L^T; ANY F with F F^T = C^-1 gives the same criterion, and the oracle
 *          takes F^T = Rc^-1 with C = Rc Rc^T (plain fp64 Cholesky of C, whitening by forward substitution: no
 *          explicit inverse).  A and y are whitened in fp64 (no rounding to fp32) and the constrained problem is
 *          solved on them; coeff_sigma is reading R3 with unit noise (the whitened noise is white: this is the
 *          projected inverse Hessian H_w itself), resid is the RMS of the WHITENED residual (dimensionless,
 *          about 1 when the model fits to the noise; reading R17 of DESIGN.md).
 *
 * Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`): brute force over every support
 * (oracle/brute.py), scaled KKT residuals recomputed in numpy, noiseless recovery, the R = 2
 * closed form, orthonormal library == Euclidean projection onto the simplex, interior case ==
 * sum-to-one closed form / unconstrained closed form, invariances,
 * Monte Carlo for the uncertainties.  The values the paper prints (0.0142, 1.2e-3, 5.5 +- 0.2 %)
 * need its real spectral library and are "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_MAX_STEPS 2000
#define ORACLE_RANK_TOL 1e-12
#define ORACLE_LAMBDA_TOL 1e-12
#define ORACLE_ROUND_TOL 1e-13

/* status bits written to status_out */
#define ORACLE_ST_OK 0
#define ORACLE_ST_RANKDEF 1     /* an index was rejected because A_F Z lost rank (R9) */
#define ORACLE_ST_STEPCAP 2     /* step cap hit: result not certified                 */
#define ORACLE_ST_NONFINITE 4   /* non-finite input: outputs NaN                      */

typedef struct {
    int L, R;
    double *y, *a, *atry, *g, *lam;        /* L, R, R, R, R */
    int *F, *inF, *blocked, *perm;          /* R each */
    double *B, *V, *Q1, *rhs, *w, *c, *Zc;  /* QR workspace */
    double *Jrow;
    int cons;                               /* 1: sum-to-one (sto, slo through the slack column); 0: pos */
} work_t;

static int work_alloc(work_t *w, int L, int R) {
    int m = R < L + 1 ? R : L + 1;          /* a support can not exceed L+1 members */
    (void)m;
    w->L = L; w->R = R; w->cons = 1;
    w->y = malloc(sizeof(double) * L);
    w->a = malloc(sizeof(double) * R);
    w->atry = malloc(sizeof(double) * R);
    w->g = malloc(sizeof(double) * R);
    w->lam = malloc(sizeof(double) * R);
    w->F = malloc(sizeof(int) * R);
    w->inF = malloc(sizeof(int) * R);
    w->blocked = malloc(sizeof(int) * R);
    w->perm = malloc(sizeof(int) * R);
    w->B = malloc(sizeof(double) * (size_t)L * R);
    w->V = malloc(sizeof(double) * (size_t)L * R);
    w->Q1 = malloc(sizeof(double) * (size_t)L * R);
    w->rhs = malloc(sizeof(double) * L);
    w->w = malloc(sizeof(double) * R);
    w->c = malloc(sizeof(double) * R);
    w->Zc = malloc(sizeof(double) * R);
    w->Jrow = malloc(sizeof(double) * R);
    return w->y && w->a && w->atry && w->g && w->lam && w->F && w->inF && w->blocked && w->perm &&
           w->B && w->V && w->Q1 && w->rhs && w->w && w->c && w->Zc && w->Jrow;
}

static void work_free(work_t *w) {
    free(w->y); free(w->a); free(w->atry); free(w->g); free(w->lam); free(w->F); free(w->inF);
    free(w->blocked); free(w->perm); free(w->B); free(w->V); free(w->Q1); free(w->rhs);
    free(w->w); free(w->c); free(w->Zc); free(w->Jrow);
}

/* Z(i, j), i = 0..k-1, j = 0..k-2: columns 2..k of the Householder reflector
 * H = I - 2 w w'/(w'w), w = u - e_1, u = 1/sqrt(k), which maps u to e_1.  H is orthogonal and
 * symmetric, H e_1 = u, so its other columns are an orthonormal basis of {z : 1'z = 0}. */
static double Zentry(int k, int i, int j) {
    double u = 1.0 / sqrt((double)k);
    double wi = u - (i == 0 ? 1.0 : 0.0);
    double wj = u;                       /* column index j+1 >= 1, so w_{j+1} = u */
    double ww = 2.0 - 2.0 * u;           /* w'w = (u-1)^2 + (k-1)u^2 = 2 - 2u */
    return ((i == j + 1) ? 1.0 : 0.0) - 2.0 * wi * wj / ww;
}

/* Column-pivoted Householder QR of B (L x m, column-major, overwritten: upper triangle = R),
 * reflector vectors kept in V (column j holds v_j, zero above row j), rhs overwritten by Q'rhs.
 * Returns the numerical rank; diag(R) magnitudes are non-increasing. */
static int qr_pivot(int L, int m, double *B, double *V, double *rhs, int *perm, double *rmin, double *rmax) {
    int rank = m;
    double r00 = 0.0;
    *rmin = INFINITY; *rmax = 0.0;
    for (int j = 0; j < m; ++j) perm[j] = j;
    for (int j = 0; j < m && j < L; ++j) {
        int p = j; double best = -1.0;
        for (int q = j; q < m; ++q) {
            double s = 0.0;
            for (int i = j; i < L; ++i) s += B[(size_t)q * L + i] * B[(size_t)q * L + i];
            if (s > best) { best = s; p = q; }
        }
        if (p != j) {
            for (int i = 0; i < L; ++i) { double t = B[(size_t)j * L + i]; B[(size_t)j * L + i] = B[(size_t)p * L + i]; B[(size_t)p * L + i] = t; }
            int t = perm[j]; perm[j] = perm[p]; perm[p] = t;
        }
        double nrm = sqrt(best);
        if (j == 0) r00 = nrm;
        if (!(nrm > ORACLE_RANK_TOL * r00) || nrm == 0.0) { rank = j; break; }
        double x0 = B[(size_t)j * L + j];
        double alpha = (x0 >= 0.0) ? -nrm : nrm;
        double *v = V + (size_t)j * L;
        for (int i = 0; i < j; ++i) v[i] = 0.0;
        for (int i = j; i < L; ++i) v[i] = B[(size_t)j * L + i];
        v[j] -= alpha;
        double vv = 0.0;
        for (int i = j; i < L; ++i) vv += v[i] * v[i];
        /* apply H = I - 2 v v'/(v'v) to the remaining columns and to rhs */
        for (int q = j + 1; q < m; ++q) {
            double s = 0.0;
            for (int i = j; i < L; ++i) s += v[i] * B[(size_t)q * L + i];
            s = 2.0 * s / vv;
            for (int i = j; i < L; ++i) B[(size_t)q * L + i] -= s * v[i];
        }
        {
            double s = 0.0;
            for (int i = j; i < L; ++i) s += v[i] * rhs[i];
            s = 2.0 * s / vv;
            for (int i = j; i < L; ++i) rhs[i] -= s * v[i];
        }
        B[(size_t)j * L + j] = alpha;
        for (int i = j + 1; i < L; ++i) B[(size_t)j * L + i] = 0.0;
        if (nrm < *rmin) *rmin = nrm;
        if (nrm > *rmax) *rmax = nrm;
    }
    if (m > L) rank = rank < L ? rank : L;
    return rank;
}

/* Equality-constrained LS on the support F (k members): returns 1 and fills atry[F] when
 * A_F Z has full column rank, 0 otherwise.  A64 is column-major (column r at A64 + r*L).
 * Leaves B (R factor), V (reflectors), perm in the workspace for the uncertainty pass. */
static int eqp_solve_free(const double *A64, work_t *w, int k, double *rmin, double *rmax);

static int eqp_solve(const double *A64, work_t *w, int k, double *rmin, double *rmax) {
    int L = w->L;
    *rmin = INFINITY; *rmax = 0.0;
    if (!w->cons) return eqp_solve_free(A64, w, k, rmin, rmax);
    if (k == 1) { w->atry[w->F[0]] = 1.0; return 1; }
    int m = k - 1;
    if (m > L) return 0;
    double a0 = 1.0 / (double)k;
    for (int l = 0; l < L; ++l) {
        double s = 0.0;
        for (int i = 0; i < k; ++i) s += A64[(size_t)w->F[i] * L + l];
        w->rhs[l] = w->y[l] - a0 * s;
    }
    for (int j = 0; j < m; ++j)
        for (int l = 0; l < L; ++l) {
            double s = 0.0;
            for (int i = 0; i < k; ++i) s += A64[(size_t)w->F[i] * L + l] * Zentry(k, i, j);
            w->B[(size_t)j * L + l] = s;
        }
    int rank = qr_pivot(L, m, w->B, w->V, w->rhs, w->perm, rmin, rmax);
    if (rank < m) return 0;
    /* back substitution R c_perm = (Q'rhs)[0:m] */
    for (int j = m - 1; j >= 0; --j) {
        double s = w->rhs[j];
        for (int q = j + 1; q < m; ++q) s -= w->B[(size_t)q * L + j] * w->w[q];
        w->w[j] = s / w->B[(size_t)j * L + j];
    }
    for (int j = 0; j < m; ++j) w->c[w->perm[j]] = w->w[j];
    for (int i = 0; i < k; ++i) {
        double s = a0;
        for (int j = 0; j < m; ++j) s += Zentry(k, i, j) * w->c[j];
        w->atry[w->F[i]] = s;
    }
    return 1;
}

/* Positivity-only sub-problem (pos option): min ||y - A_F a_F|| with no equality constraint, by column-pivoted
 * Householder QR of A_F itself.  Same workspace conventions as eqp_solve. */
static int eqp_solve_free(const double *A64, work_t *w, int k, double *rmin, double *rmax) {
    int L = w->L;
    int m = k;
    if (m > L) return 0;
    for (int l = 0; l < L; ++l) w->rhs[l] = w->y[l];
    for (int j = 0; j < m; ++j)
        for (int l = 0; l < L; ++l) w->B[(size_t)j * L + l] = A64[(size_t)w->F[j] * L + l];
    int rank = qr_pivot(L, m, w->B, w->V, w->rhs, w->perm, rmin, rmax);
    if (rank < m) return 0;
    for (int j = m - 1; j >= 0; --j) {
        double s = w->rhs[j];
        for (int q = j + 1; q < m; ++q) s -= w->B[(size_t)q * L + j] * w->w[q];
        w->w[j] = s / w->B[(size_t)j * L + j];
    }
    for (int j = 0; j < m; ++j) w->atry[w->F[w->perm[j]]] = w->w[j];
    return 1;
}

/* coeff_sigma on the final support (reading R3): a_F = a0 + Z (A_F Z)^+ (y - A_F a0), so
 * J = d a_F / d y = Z (A_F Z)^+ = Z P R^-1 Q1'  (k x L), and
 * coeff_sigma_i = sqrt( sum_l J_il^2 sigma_l^2 ); zero off the support and when k = 1.
 * Uses the QR left in the workspace by the last successful eqp_solve on this support. */
static void sigma_pass(work_t *w, int k, const float *sig, double *out) {
    int L = w->L, R = w->R;
    for (int i = 0; i < R; ++i) out[i] = 0.0;
    if (w->cons ? (k <= 1) : (k <= 0)) return;
    int m = w->cons ? k - 1 : k;           /* pos option: J = A_F^+ = P R^-1 Q1' (no Z) */
    /* Q1 = H_0 H_1 ... H_{m-1} [I_m; 0]  (L x m): apply reflectors in reverse order */
    for (int j = 0; j < m; ++j) {
        double *q = w->Q1 + (size_t)j * L;
        for (int l = 0; l < L; ++l) q[l] = (l == j) ? 1.0 : 0.0;
    }
    for (int r = m - 1; r >= 0; --r) {
        const double *v = w->V + (size_t)r * L;
        double vv = 0.0;
        for (int l = r; l < L; ++l) vv += v[l] * v[l];
        for (int j = 0; j < m; ++j) {
            double *q = w->Q1 + (size_t)j * L;
            double s = 0.0;
            for (int l = r; l < L; ++l) s += v[l] * q[l];
            s = 2.0 * s / vv;
            for (int l = r; l < L; ++l) q[l] -= s * v[l];
        }
    }
    for (int l = 0; l < L; ++l) {
        /* w = R^-1 (row l of Q1)' ; c = P w ; Jcol = Z c */
        for (int j = m - 1; j >= 0; --j) {
            double s = w->Q1[(size_t)j * L + l];
            for (int q = j + 1; q < m; ++q) s -= w->B[(size_t)q * L + j] * w->w[q];
            w->w[j] = s / w->B[(size_t)j * L + j];
        }
        for (int j = 0; j < m; ++j) w->c[w->perm[j]] = w->w[j];
        double s2 = (double)sig[l] * (double)sig[l];
        for (int i = 0; i < k; ++i) {
            double s = 0.0;
            if (w->cons) for (int j = 0; j < m; ++j) s += Zentry(k, i, j) * w->c[j];
            else s = w->c[i];
            out[w->F[i]] += s * s * s2;
        }
    }
    for (int i = 0; i < k; ++i) out[w->F[i]] = sqrt(out[w->F[i]]);
}

static double sqdist_to_column(const double *A64, const double *y, int L, int r) {
    double s = 0.0;
    for (int l = 0; l < L; ++l) { double d = y[l] - A64[(size_t)r * L + l]; s += d * d; }
    return s;
}

/* gradient g = A'(A a - y) of F/2, objective F = ||y - A a||^2 */
static double gradient(const double *A64, const work_t *w, double *g) {
    int L = w->L, R = w->R;
    double *r = w->rhs;   /* free at this point */
    for (int l = 0; l < L; ++l) r[l] = -w->y[l];
    for (int i = 0; i < R; ++i)
        if (w->a[i] != 0.0)
            for (int l = 0; l < L; ++l) r[l] += A64[(size_t)i * L + l] * w->a[i];
    double F = 0.0;
    for (int l = 0; l < L; ++l) F += r[l] * r[l];
    for (int i = 0; i < R; ++i) {
        double s = 0.0;
        for (int l = 0; l < L; ++l) s += A64[(size_t)i * L + l] * r[l];
        g[i] = s;
    }
    return F;
}

static int solve_pixel(const double *A64, work_t *w, const float *sig, double *coeffs, double *csig,
                       double *resid, double *lam_out, double *nu_out, int *k_out, int *steps_out,
                       double *rankmargin_out) {
    int L = w->L, R = w->R, status = ORACLE_ST_OK;
    for (int l = 0; l < L; ++l)
        if (!isfinite(w->y[l])) status = ORACLE_ST_NONFINITE;
    if (status == ORACLE_ST_NONFINITE) {
        for (int i = 0; i < R; ++i) { coeffs[i] = NAN; if (csig) csig[i] = NAN; if (lam_out) lam_out[i] = NAN; }
        if (resid) *resid = NAN;
        if (nu_out) *nu_out = NAN;
        if (k_out) *k_out = 0;
        if (steps_out) *steps_out = 0;
        if (rankmargin_out) *rankmargin_out = NAN;
        return status;
    }
    /* rounding scale of the gradient: s = max_i sum_l |A_li| |y_l| */
    double gscale = 0.0;
    for (int i = 0; i < R; ++i) {
        double s = 0.0;
        for (int l = 0; l < L; ++l) s += fabs(A64[(size_t)i * L + l]) * fabs(w->y[l]);
        if (s > gscale) gscale = s;
    }
    /* step 2: best vertex (pos option: the origin, which is feasible there) */
    int j0 = 0; double best = INFINITY;
    for (int i = 0; i < R; ++i) {
        double d = sqdist_to_column(A64, w->y, L, i);
        if (d < best) { best = d; j0 = i; }
    }
    for (int i = 0; i < R; ++i) { w->a[i] = 0.0; w->inF[i] = 0; w->blocked[i] = 0; w->lam[i] = 0.0; }
    int k = 1; w->F[0] = j0; w->inF[j0] = 1; w->a[j0] = 1.0;
    if (!w->cons) { k = 0; w->inF[j0] = 0; w->a[j0] = 0.0; }
    int last_added = -1, steps = 0, done = 0;
    double nu = 0.0, rmin = INFINITY, rmax = 0.0, Fobj = best;
    while (!done) {
        if (++steps > ORACLE_MAX_STEPS) { status |= ORACLE_ST_STEPCAP; break; }
        int ok = (k == 0) ? 1 : eqp_solve(A64, w, k, &rmin, &rmax);
        if (!ok) {
            /* step 3, rank-deficient: reject the index just added, block it for this pixel */
            status |= ORACLE_ST_RANKDEF;
            int rej = (last_added >= 0) ? last_added : w->F[k - 1];
            int pos = 0;
            for (int i = 0; i < k; ++i) if (w->F[i] == rej) pos = i;
            for (int i = pos; i + 1 < k; ++i) w->F[i] = w->F[i + 1];
            --k; w->inF[rej] = 0; w->blocked[rej] = 1; w->a[rej] = 0.0; last_added = -1;
            continue;
        }
        int allpos = 1;
        for (int i = 0; i < k; ++i) if (!(w->atry[w->F[i]] > 0.0)) allpos = 0;
        if (allpos) {
            /* step 4 */
            for (int i = 0; i < k; ++i) w->a[w->F[i]] = w->atry[w->F[i]];
            Fobj = gradient(A64, w, w->g);
            double gmax = 0.0;
            for (int i = 0; i < R; ++i) if (fabs(w->g[i]) > gmax) gmax = fabs(w->g[i]);
            nu = 0.0;
            if (w->cons) for (int i = 0; i < k; ++i) nu -= w->g[w->F[i]] * w->a[w->F[i]];
            int jmin = -1; double lmin = -(ORACLE_LAMBDA_TOL * gmax + ORACLE_ROUND_TOL * gscale);
            for (int i = 0; i < R; ++i) {
                w->lam[i] = w->inF[i] ? 0.0 : w->g[i] + nu;
                if (!w->inF[i] && !w->blocked[i] && w->lam[i] < lmin) { lmin = w->lam[i]; jmin = i; }
            }
            if (jmin < 0) { done = 1; break; }
            w->F[k++] = jmin; w->inF[jmin] = 1; w->a[jmin] = 0.0; last_added = jmin;
        } else {
            /* step 5: ratio step towards the sub-problem solution */
            double alpha = 1.0;
            for (int i = 0; i < k; ++i) {
                int f = w->F[i];
                if (!(w->atry[f] > 0.0)) {
                    double den = w->a[f] - w->atry[f];
                    double t = den > 0.0 ? w->a[f] / den : 0.0;
                    if (t < alpha) alpha = t;
                }
            }
            if (alpha < 0.0) alpha = 0.0;
            int nk = 0, dropped_added = 0;
            for (int i = 0; i < k; ++i) {
                int f = w->F[i];
                double an = w->a[f] + alpha * (w->atry[f] - w->a[f]);
                int blocking = !(w->atry[f] > 0.0) &&
                               (w->a[f] - w->atry[f] > 0.0 ? w->a[f] / (w->a[f] - w->atry[f]) : 0.0) <= alpha;
                if (blocking || !(an > 0.0)) {
                    w->a[f] = 0.0; w->inF[f] = 0;
                    if (f == last_added && alpha == 0.0) dropped_added = 1;
                } else {
                    w->a[f] = an; w->F[nk++] = f;
                }
            }
            if (dropped_added) w->blocked[last_added] = 1;   /* degenerate tie: do not re-add */
            k = nk; last_added = -1;
            if (w->cons) {
                if (k == 0) { status |= ORACLE_ST_STEPCAP; break; }
                /* renormalise rounding drift so that the point stays on the simplex */
                double s = 0.0;
                for (int i = 0; i < k; ++i) s += w->a[w->F[i]];
                for (int i = 0; i < k; ++i) w->a[w->F[i]] /= s;
            }
        }
    }
    for (int i = 0; i < R; ++i) coeffs[i] = w->a[i];
    if (lam_out) for (int i = 0; i < R; ++i) lam_out[i] = w->lam[i];
    if (nu_out) *nu_out = nu;
    if (resid) *resid = sqrt(Fobj / (double)L);
    if (k_out) *k_out = k;
    if (steps_out) *steps_out = steps;
    if (rankmargin_out) *rankmargin_out = (k > (w->cons ? 1 : 0)) ? rmin : INFINITY;
    if (csig) {
        if (sig) {
            int bad = 0;
            for (int l = 0; l < L; ++l) if (!isfinite(sig[l]) || !(sig[l] > 0.0f)) bad = 1;
            if (bad) for (int i = 0; i < R; ++i) csig[i] = NAN;
            else sigma_pass(w, k, sig, csig);
        } else {
            float *ones = malloc(sizeof(float) * L);
            for (int l = 0; l < L; ++l) ones[l] = 1.0f;
            sigma_pass(w, k, ones, csig);
            free(ones);
        }
    }
    return status;
}

/* Plain fp64 Cholesky C = Rc Rc' (lower), in place on the lower triangle of C (L x L, row-major).  Returns 0, or
 * -1 when C is not positive definite. */
static int cholesky_lower(double *C, int L) {
    for (int j = 0; j < L; ++j) {
        double d = C[(size_t)j * L + j];
        for (int k = 0; k < j; ++k) d -= C[(size_t)j * L + k] * C[(size_t)j * L + k];
        if (!(d > 0.0) || !isfinite(d)) return -1;
        d = sqrt(d);
        C[(size_t)j * L + j] = d;
        for (int i = j + 1; i < L; ++i) {
            double v = C[(size_t)i * L + j];
            for (int k = 0; k < j; ++k) v -= C[(size_t)i * L + k] * C[(size_t)j * L + k];
            C[(size_t)i * L + j] = v / d;
        }
    }
    return 0;
}

/* x <- Rc^-1 x (forward substitution), x has stride `inc` */
static void whiten(const double *Rc, int L, double *x, size_t inc) {
    for (int i = 0; i < L; ++i) {
        double v = x[(size_t)i * inc];
        for (int k = 0; k < i; ++k) v -= Rc[(size_t)i * L + k] * x[(size_t)k * inc];
        x[(size_t)i * inc] = v / Rc[(size_t)i * L + i];
    }
}

/*
 * Entry point.  All pointers are HOST pointers.  Layouts as include/linmin.h:
 *   A[l*R + r] float32 (L x R row-major);  Y[p*ldY + l] float32;  sigma: NULL (sigma == 1),
 *   or sigma[l] shared (sigma_stride == 0), or sigma[p*sigma_stride + l].
 *   constraint: 0 sto, 1 slo, 2 pos.  cov_kind: 0 unweighted fit; 1 diagonal covariance, cov[l] = per-channel
 *   noise STD (C = diag(cov^2)); 2 full covariance, cov[l*L + m] (symmetric positive definite).  With a
 *   covariance, sigma is ignored (the whitened noise is white) and resid is the whitened RMS.
 * Outputs (fp64; any may be NULL except coeffs): coeffs N x R, coeff_sigma N x R, resid N,
 * lambda N x R (multipliers of a >= 0, scale of g = A'(Aa - y), whitened data when weighted), nu N
 * (slo: the multiplier of sum a <= 1, >= 0; pos: 0), support_size N (non-zero coefficients),
 * steps N (active-set steps), rank_margin N (smallest |R_jj| of the final QR; INF when there is none),
 * status N (ORACLE_ST_* bits).  Returns 0, -1 on bad arguments / allocation failure, -2 when the covariance is
 * not positive definite.
 */
int linmin_oracle_solve_ex(const float *A, const float *Y, const float *sigma, int64_t N, int32_t L,
                           int32_t R, int64_t ldY, int64_t sigma_stride, int32_t constraint,
                           const float *cov, int32_t cov_kind, double *coeffs,
                           double *coeff_sigma, double *resid, double *lambda, double *nu,
                           int32_t *support_size, int32_t *steps, double *rank_margin,
                           int32_t *status, int32_t nthreads) {
    if (!A || !Y || !coeffs || N < 0 || L < 1 || R < 1) return -1;
    if (constraint < 0 || constraint > 2 || cov_kind < 0 || cov_kind > 2 || (cov_kind && !cov)) return -1;
    if (ldY == 0) ldY = L;
    if (ldY < L) return -1;
    const int Ra = (constraint == 1) ? R + 1 : R;      /* slo: the slack endmember (a zero column) comes last */
    double *A64 = calloc((size_t)L * Ra, sizeof(double));
    if (!A64) return -1;
    for (int l = 0; l < L; ++l)
        for (int r = 0; r < R; ++r) A64[(size_t)r * L + l] = (double)A[(size_t)l * R + r];
    double *Rc = NULL;
    float *ones = NULL;
    if (cov_kind) {
        Rc = calloc((size_t)L * L, sizeof(double));
        ones = malloc(sizeof(float) * L);
        if (!Rc || !ones) { free(A64); free(Rc); free(ones); return -1; }
        for (int l = 0; l < L; ++l) ones[l] = 1.0f;
        if (cov_kind == 1) {
            for (int l = 0; l < L; ++l) Rc[(size_t)l * L + l] = (double)cov[l] * (double)cov[l];
        } else {
            for (int l = 0; l < L; ++l)
                for (int m = 0; m <= l; ++m) Rc[(size_t)l * L + m] = 0.5 * ((double)cov[(size_t)l * L + m] + (double)cov[(size_t)m * L + l]);
        }
        if (cholesky_lower(Rc, L) != 0) { free(A64); free(Rc); free(ones); return -2; }
        for (int r = 0; r < R; ++r) whiten(Rc, L, A64 + (size_t)r * L, 1);      /* S' = S.L of eq. 6 */
    }
    int fail = 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel
    {
        work_t w;
        int okw = work_alloc(&w, L, Ra);
        double *ca = okw ? malloc(sizeof(double) * 3 * (size_t)Ra) : NULL;    /* coeffs, sigma, lambda of the augmented problem */
        if (!okw || !ca) {
            okw = 0;
#pragma omp atomic write
            fail = 1;
        }
        if (okw) w.cons = (constraint != 2);
#pragma omp for schedule(dynamic, 64)
        for (int64_t p = 0; p < N; ++p) {
            if (!okw) continue;
            for (int l = 0; l < L; ++l) w.y[l] = (double)Y[p * ldY + l];
            if (cov_kind) {
                int finite = 1;
                for (int l = 0; l < L; ++l) if (!isfinite(w.y[l])) finite = 0;
                if (finite) whiten(Rc, L, w.y, 1);                              /* X' = X.L of eq. 6 */
            }
            const float *sig = cov_kind ? ones : (sigma ? sigma + p * sigma_stride : NULL);
            int32_t kk = 0, st = 0; double rm = 0.0;
            double *cp = (Ra == R) ? coeffs + p * R : ca;
            double *sp = coeff_sigma ? ((Ra == R) ? coeff_sigma + p * R : ca + Ra) : NULL;
            double *lp = lambda ? ((Ra == R) ? lambda + p * R : ca + 2 * Ra) : NULL;
            int s = solve_pixel(A64, &w, sig, cp, sp, resid ? resid + p : NULL, lp,
                                nu ? nu + p : NULL, &kk, &st, &rm);
            if (Ra != R) {      /* slo: drop the slack column; it does not count as a member of the support */
                for (int i = 0; i < R; ++i) coeffs[p * R + i] = ca[i];
                if (coeff_sigma) for (int i = 0; i < R; ++i) coeff_sigma[p * R + i] = ca[Ra + i];
                if (lambda) for (int i = 0; i < R; ++i) lambda[p * R + i] = ca[2 * Ra + i];
                if (ca[R] > 0.0) --kk;
            }
            if (support_size) support_size[p] = kk;
            if (steps) steps[p] = st;
            if (rank_margin) rank_margin[p] = rm;
            if (status) status[p] = s;
        }
        if (okw) work_free(&w);
        free(ca);
    }
    free(A64); free(Rc); free(ones);
    return fail ? -1 : 0;
}

/* The hot path: sum-to-one, unweighted. */
int linmin_oracle_solve(const float *A, const float *Y, const float *sigma, int64_t N, int32_t L,
                        int32_t R, int64_t ldY, int64_t sigma_stride, double *coeffs,
                        double *coeff_sigma, double *resid, double *lambda, double *nu,
                        int32_t *support_size, int32_t *steps, double *rank_margin,
                        int32_t *status, int32_t nthreads) {
    return linmin_oracle_solve_ex(A, Y, sigma, N, L, R, ldY, sigma_stride, 0, NULL, 0, coeffs, coeff_sigma, resid,
                                  lambda, nu, support_size, steps, rank_margin, status, nthreads);
}

int linmin_oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

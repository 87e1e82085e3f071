/*
 * bj_oracle.c -- TEST INFRASTRUCTURE, not the product.
 *
 * A plain, slow, obviously-correct fp64 CPU statement of the block-Jacobi preconditioning
 * path of arxiv 2410.02408, written from the paper (citations are PAPER.md line numbers)
 * and from the readings of SURVEY.md section 8(c).  It shares no code, header, table or
 * helper with the CUDA library under paper_2410_02408_b200/csrc/.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * Build: gcc -O2 -ffp-contract=off -fPIC -shared [-fopenmp] bj_oracle.c -o libbj_oracle.so -lm
 *   -ffp-contract=off: every multiply and add rounds separately, exactly as written.
 *   OpenMP (optional) only distributes INDEPENDENT rows / blocks over threads; no
 *   floating-point sum is ever split across threads, so results are identical with
 *   and without it.  Dot products and norms are serial left-to-right sums.
 *
 * Pins (tests/test_oracle_pins.py): closed-form Laplacian spectra, line-block spectra,
 * b=N => identity, block-diagonal model of PAPER.md:80, numpy/scipy library routines on
 * random SPD blocks, dense eigensolves for N<=1024, m=N Lanczos == dense spectrum.
 * PCG (orc_pcg): numpy dense solve, scipy.sparse.linalg.cg iterates, M = A => one step, CG-Lanczos Ritz values.
 * Unpinned against truth: kappa estimates of the five full-size configs (no closed form);
 * those are pinned only by the invariants above.  See DESIGN.md section 3.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_OK 0
#define ORC_NOT_SPD (-4)
#define ORC_ALLOC (-5)

/* ---- step 1: y = A x, CSR, left-to-right within a row ------------- */
void orc_spmv(int64_t n, const int32_t* rp, const int32_t* ci, const double* val,
              const double* x, double* y)
{
    int64_t i;
#pragma omp parallel for schedule(static)
    for (i = 0; i < n; ++i) {
        double s = 0.0;
        for (int32_t p = rp[i]; p < rp[i + 1]; ++p) s += val[p] * x[ci[p]];
        y[i] = s;
    }
}

/* ---- step 2: diagonal-block extraction (sec 3.2; listing 191-197) -------
 * Block k covers indices [k b, min((k+1) b, n)).  D is nblocks x b x b row-major, zero
 * where A stores nothing; a ragged last block uses only its leading nb x nb corner.       */
void orc_extract(int64_t n, const int32_t* rp, const int32_t* ci, const double* val,
                 int64_t b, double* D)
{
    int64_t nblocks = (n + b - 1) / b;
    int64_t k;
#pragma omp parallel for schedule(static)
    for (k = 0; k < nblocks; ++k) {
        int64_t lo = k * b, hi = lo + b < n ? lo + b : n;
        double* Dk = D + k * b * b;
        for (int64_t e = 0; e < b * b; ++e) Dk[e] = 0.0;
        for (int64_t i = lo; i < hi; ++i)
            for (int32_t p = rp[i]; p < rp[i + 1]; ++p) {
                int64_t j = ci[p];
                if (j >= lo && j < hi) Dk[(i - lo) * b + (j - lo)] = val[p];
            }
    }
}

/* ---- step 3: unblocked lower Cholesky D = L L^T of one nb x nb block with leading
 * dimension ld; reads only the lower triangle; returns 1 if a radicand is <= 0 or NaN.
 * b = 1 is the paper's kernel M[i] = 1/A[i][i] in split form L = sqrt(a_ii). */
static int chol_block(double* D, int64_t nb, int64_t ld)
{
    for (int64_t j = 0; j < nb; ++j) {
        double s = D[j * ld + j];
        for (int64_t p = 0; p < j; ++p) s -= D[j * ld + p] * D[j * ld + p];
        if (!(s > 0.0) || isinf(s)) return 1;
        double ljj = sqrt(s);
        D[j * ld + j] = ljj;
        for (int64_t i = j + 1; i < nb; ++i) {
            double t = D[i * ld + j];
            for (int64_t p = 0; p < j; ++p) t -= D[i * ld + p] * D[j * ld + p];
            D[i * ld + j] = t / ljj;
        }
    }
    for (int64_t i = 0; i < nb; ++i)            /* make the strict upper triangle zero */
        for (int64_t j = i + 1; j < nb; ++j) D[i * ld + j] = 0.0;
    return 0;
}

/* factor all blocks in place; returns ORC_OK or ORC_NOT_SPD with *bad_block = first failing block */
int orc_factor(int64_t n, int64_t b, double* D, int64_t* bad_block)
{
    int64_t nblocks = (n + b - 1) / b;
    int64_t bad = nblocks;
    int64_t k;
#pragma omp parallel for schedule(static)
    for (k = 0; k < nblocks; ++k) {
        int64_t lo = k * b, hi = lo + b < n ? lo + b : n;
        if (chol_block(D + k * b * b, hi - lo, b)) {
#pragma omp critical
            { if (k < bad) bad = k; }
        }
    }
    if (bad_block) *bad_block = bad < nblocks ? bad : -1;
    return bad < nblocks ? ORC_NOT_SPD : ORC_OK;
}

/* ---- step 4: y = L^-1 r (forward) and x = L^-T y (backward), block by block ------------- */
void orc_solve_L(int64_t n, int64_t b, const double* L, const double* r, double* y)
{
    int64_t nblocks = (n + b - 1) / b;
    int64_t k;
#pragma omp parallel for schedule(static)
    for (k = 0; k < nblocks; ++k) {
        int64_t lo = k * b, hi = lo + b < n ? lo + b : n, nb = hi - lo;
        const double* Lk = L + k * b * b;
        for (int64_t i = 0; i < nb; ++i) {
            double s = r[lo + i];
            for (int64_t j = 0; j < i; ++j) s -= Lk[i * b + j] * y[lo + j];
            y[lo + i] = s / Lk[i * b + i];
        }
    }
}

void orc_solve_Lt(int64_t n, int64_t b, const double* L, const double* y, double* x)
{
    int64_t nblocks = (n + b - 1) / b;
    int64_t k;
#pragma omp parallel for schedule(static)
    for (k = 0; k < nblocks; ++k) {
        int64_t lo = k * b, hi = lo + b < n ? lo + b : n, nb = hi - lo;
        const double* Lk = L + k * b * b;
        for (int64_t i = nb - 1; i >= 0; --i) {
            double s = y[lo + i];
            for (int64_t j = i + 1; j < nb; ++j) s -= Lk[j * b + i] * x[lo + j];
            x[lo + i] = s / Lk[i * b + i];
        }
    }
}

/* ---- step 5: z = M^-1 r = L^-T (L^-1 r)  (b~ = M b of PAPER.md:88-90, M = blockdiag(D_k)) and
 * y = L^-1 A L^-T x (symmetric split form of A~ = M A; SURVEY 8(c) reading 1).
 * b == 0 means no preconditioner: op_apply = spmv.  tmp has 2 n doubles.                   */
void orc_apply(int64_t n, int64_t b, const double* L, const double* r, double* z, double* tmp)
{
    orc_solve_L(n, b, L, r, tmp);
    orc_solve_Lt(n, b, L, tmp, z);
}

void orc_op_apply(int64_t n, const int32_t* rp, const int32_t* ci, const double* val,
                  int64_t b, const double* L, const double* x, double* y, double* tmp)
{
    if (b == 0) { orc_spmv(n, rp, ci, val, x, y); return; }
    double* t = tmp;
    double* u = tmp + n;
    orc_solve_Lt(n, b, L, x, t);
    orc_spmv(n, rp, ci, val, t, u);
    orc_solve_L(n, b, L, u, y);
}

/* ---- seeded start vector (SURVEY 8(c) reading 10): integer mixer, exact int->double ----- */
static uint64_t mix64(uint64_t seed, uint64_t i)
{
    uint64_t z = seed + (i + 1u) * 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

void orc_seeded_vector(uint64_t seed, int64_t n, double* v)
{
    for (int64_t i = 0; i < n; ++i) {
        double u = (double)(mix64(seed, (uint64_t)i) >> 11) * (1.0 / 9007199254740992.0);
        v[i] = 2.0 * u - 1.0;
    }
}

/* ---- step 6: Lanczos on op = L^-1 A L^-T (or A when b == 0) -------
 *   v_1 = v0/||v0||, v_0 = 0, beta_1 = 0
 *   for j = 1..m:  w = op(v_j) - beta_j v_{j-1};  alpha_j = v_j^T w;  w -= alpha_j v_j;
 *                  if reorth: twice { c = V_j^T w; w -= V_j c } over all stored v_1..v_j;
 *                  beta_{j+1} = ||w||;  stop (m_eff = j) if beta_{j+1} <= tol_bd max_i |alpha_i|;
 *                  v_{j+1} = w / beta_{j+1}
 * alpha[0..m_eff-1] = alpha_1.., beta[0..m_eff-1] = beta_2..beta_{m_eff+1}
 * (beta[j-1] couples v_j and v_{j+1}; the last one is the residual norm).                  */
static double dot(int64_t n, const double* a, const double* b)
{
    double s = 0.0;
    for (int64_t i = 0; i < n; ++i) s += a[i] * b[i];
    return s;
}

int orc_lanczos(int64_t n, const int32_t* rp, const int32_t* ci, const double* val,
                int64_t b, const double* L, const double* v0, int m, int reorth, double tol_bd,
                double* alpha, double* beta, int* m_eff)
{
    int keep = reorth ? m : 2;
    double* V = (double*)malloc((size_t)keep * (size_t)n * sizeof(double));
    double* w = (double*)malloc((size_t)n * sizeof(double));
    double* tmp = (double*)malloc((size_t)2 * (size_t)n * sizeof(double));
    double* c = (double*)malloc((size_t)(m + 1) * sizeof(double));
    if (!V || !w || !tmp || !c) { free(V); free(w); free(tmp); free(c); return ORC_ALLOC; }
#define VCOL(j) (V + (size_t)(reorth ? (j) : ((j) & 1)) * (size_t)n)   /* v_{j+1} lives in column j */
    double nrm = sqrt(dot(n, v0, v0));
    for (int64_t i = 0; i < n; ++i) VCOL(0)[i] = v0[i] / nrm;
    double beta_j = 0.0, amax = 0.0;
    int done = 0;
    for (int j = 0; j < m; ++j) {
        double* vj = VCOL(j);
        orc_op_apply(n, rp, ci, val, b, L, vj, w, tmp);
        if (j > 0) {
            const double* vp = VCOL(j - 1);
            for (int64_t i = 0; i < n; ++i) w[i] -= beta_j * vp[i];
        }
        double a = dot(n, vj, w);
        for (int64_t i = 0; i < n; ++i) w[i] -= a * vj[i];
        if (reorth)
            for (int pass = 0; pass < 2; ++pass) {
                for (int q = 0; q <= j; ++q) c[q] = dot(n, VCOL(q), w);
                for (int q = 0; q <= j; ++q) {
                    const double* vq = VCOL(q);
                    double cq = c[q];
                    for (int64_t i = 0; i < n; ++i) w[i] -= cq * vq[i];
                }
            }
        double bn = sqrt(dot(n, w, w));
        alpha[j] = a;
        beta[j] = bn;
        done = j + 1;
        if (fabs(a) > amax) amax = fabs(a);
        if (!(bn > tol_bd * amax)) break;             /* breakdown: invariant subspace found */
        if (j + 1 < m) {
            double* vn = VCOL(j + 1);
            for (int64_t i = 0; i < n; ++i) vn[i] = w[i] / bn;
        }
        beta_j = bn;
    }
#undef VCOL
    *m_eff = done;
    free(V); free(w); free(tmp); free(c);
    return ORC_OK;
}

/* ---- step 7: extreme eigenvalues of T = tridiag(off; diag) by Sturm-sequence bisection ---
 * diag[0..m-1] = alpha, off[0..m-2] = beta coupling rows i and i+1.
 * count(x) = number of eigenvalues < x = number of negative pivots of T - x I.             */
static int sturm_count(int m, const double* d, const double* e, double x)
{
    int cnt = 0;
    double q = d[0] - x;
    if (q < 0.0) ++cnt;
    for (int i = 1; i < m; ++i) {
        double den = q;
        if (den == 0.0) den = 1e-300;
        q = (d[i] - x) - e[i - 1] * e[i - 1] / den;
        if (q < 0.0) ++cnt;
    }
    return cnt;
}

static double kth_eigenvalue(int m, const double* d, const double* e, int k)
{
    /* Gershgorin interval, then bisect until the interval cannot shrink in fp64 */
    double lo = d[0], hi = d[0];
    for (int i = 0; i < m; ++i) {
        double r = (i > 0 ? fabs(e[i - 1]) : 0.0) + (i + 1 < m ? fabs(e[i]) : 0.0);
        if (d[i] - r < lo) lo = d[i] - r;
        if (d[i] + r > hi) hi = d[i] + r;
    }
    for (int it = 0; it < 2000; ++it) {
        double mid = lo + 0.5 * (hi - lo);
        if (!(mid > lo && mid < hi)) break;
        if (sturm_count(m, d, e, mid) > k) hi = mid; else lo = mid;
    }
    return lo + 0.5 * (hi - lo);
}

/* last component of the unit eigenvector of T for eigenvalue theta, by the twisted
 * factorisation (Parlett & Dhillon): top-down pivots dp, bottom-up pivots dm,
 * gamma_k = dp_k + dm_k - (d_k - theta); twist at the k minimising |gamma_k|; then
 * z_k = 1, z_i = -e_i z_{i+1} / dp_i (i < k), z_i = -e_{i-1} z_{i-1} / dm_i (i > k).       */
static double last_component(int m, const double* d, const double* e, double theta)
{
    if (m == 1) return 1.0;
    double* dp = (double*)malloc((size_t)m * sizeof(double));
    double* dm = (double*)malloc((size_t)m * sizeof(double));
    double* z = (double*)malloc((size_t)m * sizeof(double));
    const double tiny = 1e-300;
    dp[0] = d[0] - theta;
    for (int i = 1; i < m; ++i) {
        double den = dp[i - 1] == 0.0 ? tiny : dp[i - 1];
        dp[i] = (d[i] - theta) - e[i - 1] * e[i - 1] / den;
    }
    dm[m - 1] = d[m - 1] - theta;
    for (int i = m - 2; i >= 0; --i) {
        double den = dm[i + 1] == 0.0 ? tiny : dm[i + 1];
        dm[i] = (d[i] - theta) - e[i] * e[i] / den;
    }
    int k = 0;
    double gbest = INFINITY;
    for (int i = 0; i < m; ++i) {
        double g = fabs(dp[i] + dm[i] - (d[i] - theta));
        if (g < gbest) { gbest = g; k = i; }
    }
    z[k] = 1.0;
    for (int i = k - 1; i >= 0; --i) z[i] = -e[i] * z[i + 1] / (dp[i] == 0.0 ? tiny : dp[i]);
    for (int i = k + 1; i < m; ++i) z[i] = -e[i - 1] * z[i - 1] / (dm[i] == 0.0 ? tiny : dm[i]);
    double nrm2 = 0.0;
    for (int i = 0; i < m; ++i) nrm2 += z[i] * z[i];
    double last = fabs(z[m - 1]) / sqrt(nrm2);
    free(dp); free(dm); free(z);
    return last;
}

/* m = m_eff; alpha[0..m-1]; beta[0..m-1] (beta[m-1] = beta_{m+1}, the residual norm).
 * out: theta_min, theta_max, and the Ritz residual bounds beta_{m+1} |s_{m,i}|.           */
void orc_tridiag_extremes(int m, const double* alpha, const double* beta,
                          double* tmin, double* tmax, double* res_min, double* res_max)
{
    *tmin = kth_eigenvalue(m, alpha, beta, 0);
    *tmax = kth_eigenvalue(m, alpha, beta, m - 1);
    if (res_min) *res_min = fabs(beta[m - 1]) * last_component(m, alpha, beta, *tmin);
    if (res_max) *res_max = fabs(beta[m - 1]) * last_component(m, alpha, beta, *tmax);
}

/* all eigenvalues of the tridiagonal by bisection (tests: m = N Ritz values vs dense spectrum) */
void orc_tridiag_all(int m, const double* alpha, const double* beta, double* out)
{
    for (int k = 0; k < m; ++k) out[k] = kth_eigenvalue(m, alpha, beta, k);
}

/* ---- NEXT-1: preconditioned conjugate gradients, the classical stand-in for the solve
 * stage that follows the preconditioning path, with M = blockdiag(D_k) = L L^T applied
 * as z = M^-1 r (b~ = M b) and the paper's accuracy metric ||Ax - b|| / ||b||
 * (threshold 1e-3 at PAPER.md:388).  Textbook Hestenes-Stiefel ordering, x_0 = 0:
 *   r = b; z = M^-1 r; p = z; rho = r.z
 *   repeat: q = A p; a = rho / (p.q); x += a p; r -= a q; stop if ||r|| / ||b|| <= rtol;
 *           z = M^-1 r; rho' = r.z; bt = rho' / rho; p = z + bt p; rho = rho'
 * alpha[k] = a_k, beta[k] = bt_k (one fewer than alpha when the loop stops on rtol), relres[k] = ||r_{k+1}|| / ||b||
 * from the recurrence; *true_relres = ||A x - b|| / ||b|| recomputed from x.  b == 0: M = I.                   */
int orc_pcg(int64_t n, const int32_t* rp, const int32_t* ci, const double* val, int64_t b, const double* L,
            const double* rhs, double* x, int max_iters, double rtol, double* alpha, double* beta,
            double* relres, int* iters, double* true_relres)
{
    double* r = (double*)malloc((size_t)n * sizeof(double));
    double* z = (double*)malloc((size_t)n * sizeof(double));
    double* p = (double*)malloc((size_t)n * sizeof(double));
    double* q = (double*)malloc((size_t)n * sizeof(double));
    double* tmp = (double*)malloc((size_t)2 * (size_t)n * sizeof(double));
    if (!r || !z || !p || !q || !tmp) { free(r); free(z); free(p); free(q); free(tmp); return ORC_ALLOC; }
    const double bnorm = sqrt(dot(n, rhs, rhs));
    for (int64_t i = 0; i < n; ++i) { x[i] = 0.0; r[i] = rhs[i]; }
    *iters = 0;
    *true_relres = 0.0;
    if (bnorm > 0.0) {
        if (b > 0) orc_apply(n, b, L, r, z, tmp); else memcpy(z, r, (size_t)n * sizeof(double));
        memcpy(p, z, (size_t)n * sizeof(double));
        double rho = dot(n, r, z);
        for (int k = 0; k < max_iters; ++k) {
            orc_spmv(n, rp, ci, val, p, q);
            const double a = rho / dot(n, p, q);
            for (int64_t i = 0; i < n; ++i) x[i] += a * p[i];
            for (int64_t i = 0; i < n; ++i) r[i] -= a * q[i];
            alpha[k] = a;
            relres[k] = sqrt(dot(n, r, r)) / bnorm;
            *iters = k + 1;
            if (relres[k] <= rtol) break;
            if (b > 0) orc_apply(n, b, L, r, z, tmp); else memcpy(z, r, (size_t)n * sizeof(double));
            const double rho_new = dot(n, r, z);
            const double bt = rho_new / rho;
            beta[k] = bt;
            for (int64_t i = 0; i < n; ++i) p[i] = z[i] + bt * p[i];
            rho = rho_new;
        }
        orc_spmv(n, rp, ci, val, x, q);
        double s = 0.0;
        for (int64_t i = 0; i < n; ++i) { const double d = q[i] - rhs[i]; s += d * d; }
        *true_relres = sqrt(s) / bnorm;
    }
    free(r); free(z); free(p); free(q); free(tmp);
    return ORC_OK;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}

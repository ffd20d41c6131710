/*
 * tbpm_oracle.c -- ORACLE: plain, slow, obviously-correct CPU statement of the TBPM hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.  It shares no code, header, table or
 * helper with the CUDA library (paper_2509_26309_b200/csrc) and neither includes the other.
 *
 * What it computes (SURVEY.md section 8(c) "Algorithm (authoritative statement)"; passages of
 * /root/reference/PAPER.md cited at each function):
 *
 *   tau = s*dt;  K = min{k >= ceil(tau): |J_k(tau)| < tol};  c_0 = J_0(tau), c_k = 2 (-i)^k J_k(tau)
 *   for each state:  psi = psi_start
 *     for n = 1..n_step:
 *        p0 = psi; p1 = (1/s) H p0; wf_out = c_0 p0 + c_1 p1
 *        for k = 2..K-1:  p2 = p0;  amxsy(2/s, p1, p0)  [p0 <- (2/s) H p1 - p0];  axpy(c_k, p2, wf_out);
 *                         p0 = p1; p1 = p2                                  (section 2.2.1)
 *        psi = wf_out;  corr[n-1] = <psi0|psi>;  norm2[n-1] = <psi|psi>
 *
 * Precision: fp64 (complex128, as the paper's solver, PAPER.md:1733 and BASELINE.json), Bessel functions and
 * the two dot products accumulated in long double (reading #26).  No blocking, fusion or reordering beyond
 * the loop the paper prints.
 *
 * Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): Bessel values/sum rules, Jacobi-Anger closed form,
 * K(pi)=21, exact diagonalisation (numpy.linalg.eigh) on N<=512 models of all three lattices, dimer closed
 * form, eigenstate closed forms, clean-cubic LDOS closed form g_n^3, semigroup and prefix properties, norm,
 * brute-force dense H for the CSR builder, closed-form honeycomb / chain DOS.  Nothing here is "parity
 * unpinned".
 *
 * Build: gcc -O2 -std=c11 -fopenmp -shared -fPIC tbpm_oracle.c -o libtbpm_oracle.so -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_EINVAL (-1)
#define ORACLE_ENOMEM (-2)

/* ---------------------------------------------------------------------------------------------------------
 * Bessel functions of the first kind J_0..J_kmax at x >= 0.
 * [paper silent; reading #2]  Miller's backward recurrence J_{k-1} = (2k/x) J_k - J_{k+1} started far above
 * max(kmax, x), normalised with the sum rule J_0 + 2 sum_{k>=1} J_{2k} = 1, in long double.
 * ------------------------------------------------------------------------------------------------------- */
int oracle_bessel_j(double x, int kmax, double *J)
{
    if (kmax < 0 || !J || !(x >= 0.0) || !isfinite(x)) return ORACLE_EINVAL;
    if (x == 0.0) {
        J[0] = 1.0;
        for (int k = 1; k <= kmax; ++k) J[k] = 0.0;
        return ORACLE_OK;
    }
    int top = (kmax > (int)x ? kmax : (int)x) + 60 + (int)(4.0 * sqrt(x + (double)kmax + 1.0));
    if (top & 1) ++top;                         /* even start */
    long double *j = (long double *)malloc(sizeof(long double) * (size_t)(top + 2));
    if (!j) return ORACLE_ENOMEM;
    j[top + 1] = 0.0L;
    j[top] = 1e-300L;
    for (int k = top; k >= 1; --k) {
        j[k - 1] = (2.0L * (long double)k / (long double)x) * j[k] - j[k + 1];
        if (fabsl(j[k - 1]) > 1e+1000L) {       /* rescale everything computed so far */
            for (int m = k - 1; m <= top; ++m) j[m] *= 1e-1000L;
        }
    }
    long double norm = j[0];
    for (int k = 2; k <= top; k += 2) norm += 2.0L * j[k];
    for (int k = 0; k <= kmax; ++k) J[k] = (double)(j[k] / norm);
    free(j);
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------------------
 * Chebyshev coefficients of exp(-i tau x) on [-1,1]:  c_k = (2 - delta_k0) (-i)^k J_k(tau)
 * ("the imaginary factor ... has been merged into the Chebyshev coefficients", PAPER.md:434;
 *  formula and truncation |J_k| < 1e-15 from BASELINE.json:configs[0]; readings #1, #3).
 * K = first k >= ceil(tau) with |J_k(tau)| < tol (strict);  terms k = 0..K-1 are kept.
 * coeff is [kcap][2] (re, im).  Returns K via *K_out; ORACLE_ENOMEM if K > kcap.
 * ------------------------------------------------------------------------------------------------------- */
int oracle_cheb_coeff(double tau, double tol, int kcap, int *K_out, double *coeff)
{
    if (!(tau >= 0.0) || !isfinite(tau) || !(tol > 0.0) || kcap < 1 || !K_out || !coeff) return ORACLE_EINVAL;
    int kmax = (int)ceil(tau) + 64 + (int)(8.0 * cbrt(tau + 1.0));
    double *J = (double *)malloc(sizeof(double) * (size_t)(kmax + 1));
    if (!J) return ORACLE_ENOMEM;
    int rc = oracle_bessel_j(tau, kmax, J);
    if (rc) { free(J); return rc; }
    int K = -1;
    for (int k = (int)ceil(tau); k <= kmax; ++k)
        if (fabs(J[k]) < tol) { K = k; break; }
    if (K < 1) { free(J); return ORACLE_EINVAL; }   /* tau == 0 gives K = 1 (J_0 = 1 kept, J_1 = 0 dropped) */
    if (K > kcap) { free(J); *K_out = K; return ORACLE_ENOMEM; }
    for (int k = 0; k < K; ++k) {
        double m = (k == 0 ? 1.0 : 2.0) * J[k];
        switch (k & 3) {                        /* (-i)^k = 1, -i, -1, +i */
        case 0: coeff[2 * k] = m;   coeff[2 * k + 1] = 0.0; break;
        case 1: coeff[2 * k] = 0.0; coeff[2 * k + 1] = -m;  break;
        case 2: coeff[2 * k] = -m;  coeff[2 * k + 1] = 0.0; break;
        default: coeff[2 * k] = 0.0; coeff[2 * k + 1] = m;  break;
        }
    }
    *K_out = K;
    free(J);
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------------------
 * Canonical CSR of H from the hopping list (readings #13-#17).
 *   entry (i, j, v)  =>  H[i][j] = v  and  H[j][i] = conj(v)      (<i,0|H|j,R>)
 *   hops_full != 0   =>  the list already holds both orientations; no conjugate partner is added
 *   onsite != NULL   =>  a diagonal entry (onsite_i, 0) for EVERY row (on-site energy is an orbital attribute,
 *                        PAPER.md:754-756; a hop with i == j is illegal)
 * Rows ascending, columns strictly ascending within a row.  Counting sort by row, then insertion sort of
 * each row by column.  rowptr[n_orb+1] int64, col[nnz] int32, val[nnz][2].
 * Returns ORACLE_EINVAL for an out-of-range index, a diagonal hop, or a duplicate (row, col).
 * ------------------------------------------------------------------------------------------------------- */
int oracle_build_csr(int64_t n_orb, const double *onsite, int64_t n_hop, const int32_t *hop_i, const int32_t *hop_j,
                     const double *hop_val, int hops_full, int64_t *rowptr, int32_t *col, double *val)
{
    if (n_orb < 0 || n_hop < 0 || !rowptr) return ORACLE_EINVAL;
    for (int64_t r = 0; r <= n_orb; ++r) rowptr[r] = 0;
    for (int64_t h = 0; h < n_hop; ++h) {
        int32_t i = hop_i[h], j = hop_j[h];
        if (i < 0 || j < 0 || i >= n_orb || j >= n_orb || i == j) return ORACLE_EINVAL;
        rowptr[i + 1]++;
        if (!hops_full) rowptr[j + 1]++;
    }
    if (onsite) for (int64_t r = 0; r < n_orb; ++r) rowptr[r + 1]++;
    for (int64_t r = 0; r < n_orb; ++r) rowptr[r + 1] += rowptr[r];
    int64_t *fill = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n_orb + 1));
    if (!fill) return ORACLE_ENOMEM;
    memcpy(fill, rowptr, sizeof(int64_t) * (size_t)(n_orb + 1));
    if (onsite) for (int64_t r = 0; r < n_orb; ++r) {
        int64_t p = fill[r]++;
        col[p] = (int32_t)r; val[2 * p] = onsite[r]; val[2 * p + 1] = 0.0;
    }
    for (int64_t h = 0; h < n_hop; ++h) {
        int32_t i = hop_i[h], j = hop_j[h];
        int64_t p = fill[i]++;
        col[p] = j; val[2 * p] = hop_val[2 * h]; val[2 * p + 1] = hop_val[2 * h + 1];
        if (!hops_full) {
            int64_t q = fill[j]++;
            col[q] = i; val[2 * q] = hop_val[2 * h]; val[2 * q + 1] = -hop_val[2 * h + 1];
        }
    }
    free(fill);
    for (int64_t r = 0; r < n_orb; ++r) {
        for (int64_t p = rowptr[r] + 1; p < rowptr[r + 1]; ++p) {
            int32_t c = col[p]; double vr = val[2 * p], vi = val[2 * p + 1];
            int64_t q = p - 1;
            while (q >= rowptr[r] && col[q] > c) {
                col[q + 1] = col[q]; val[2 * q + 2] = val[2 * q]; val[2 * q + 3] = val[2 * q + 1]; --q;
            }
            col[q + 1] = c; val[2 * q + 2] = vr; val[2 * q + 3] = vi;
        }
        for (int64_t p = rowptr[r] + 1; p < rowptr[r + 1]; ++p)
            if (col[p] == col[p - 1]) return ORACLE_EINVAL;     /* duplicate pair (reading #15) */
    }
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------------------
 * amxsy on the hopping list, serial scatter form (AUTHORITATIVE):  y <- a*H*x - y   (sub != 0)
 *                                                                  y <- a*H*x       (sub == 0)
 * "amxsy defined as y = aMx - y with a being a real number".
 * (H x)[i] = onsite[i] x[i] + sum_{h: i_h = i} v_h x[j_h] + sum_{h: j_h = i} conj(v_h) x[i_h]
 * ------------------------------------------------------------------------------------------------------- */
static void amxsy_hops(int64_t n_orb, const double *onsite, int64_t n_hop, const int32_t *hop_i, const int32_t *hop_j,
                       const double *hop_val, int hops_full, double a, const double *x, double *y, int sub)
{
    for (int64_t i = 0; i < n_orb; ++i) {
        double d = onsite ? a * onsite[i] : 0.0;
        double yr = d * x[2 * i], yi = d * x[2 * i + 1];
        if (sub) { yr -= y[2 * i]; yi -= y[2 * i + 1]; }
        y[2 * i] = yr; y[2 * i + 1] = yi;
    }
    for (int64_t h = 0; h < n_hop; ++h) {
        int64_t i = hop_i[h], j = hop_j[h];
        double vr = a * hop_val[2 * h], vi = a * hop_val[2 * h + 1];
        /* y[i] += v * x[j] */
        y[2 * i]     += vr * x[2 * j] - vi * x[2 * j + 1];
        y[2 * i + 1] += vr * x[2 * j + 1] + vi * x[2 * j];
        if (!hops_full) {                       /* y[j] += conj(v) * x[i] */
            y[2 * j]     += vr * x[2 * i] + vi * x[2 * i + 1];
            y[2 * j + 1] += vr * x[2 * i + 1] - vi * x[2 * i];
        }
    }
}

/* y <- y + c*x, complex c   ("axpy is y = ax + y") */
static void axpy_c(int64_t n, double cr, double ci, const double *x, double *y)
{
    for (int64_t i = 0; i < n; ++i) {
        y[2 * i]     += cr * x[2 * i] - ci * x[2 * i + 1];
        y[2 * i + 1] += cr * x[2 * i + 1] + ci * x[2 * i];
    }
}

/* <a|b> = sum_i conj(a_i) b_i and <b|b>, long double accumulation (reading #26) */
static void dots(int64_t n, const double *a, const double *b, double *corr_re, double *corr_im, double *norm2)
{
    long double sr = 0.0L, si = 0.0L, nn = 0.0L;
    for (int64_t i = 0; i < n; ++i) {
        long double ar = a[2 * i], ai = a[2 * i + 1], br = b[2 * i], bi = b[2 * i + 1];
        sr += ar * br + ai * bi;
        si += ar * bi - ai * br;
        nn += br * br + bi * bi;
    }
    *corr_re = (double)sr; *corr_im = (double)si; *norm2 = (double)nn;
}

/* ---------------------------------------------------------------------------------------------------------
 * One state, n_step time steps (calc_corr_dos for one random sample; one independent
 * propagation per initial state).
 *   psi_start [n_orb][2]  state at the start of the window (= psi0 for a run from t = 0)
 *   psi0      [n_orb][2]  bra of the correlation  corr_n = <psi0|psi(t_n)>
 *   corr [n_step][2], norm2 [n_step] (may be NULL), psi_final [n_orb][2] (may be NULL)
 * corr[n] is t = (n+1)*dt after psi_start (reading #7).
 * ------------------------------------------------------------------------------------------------------- */
int oracle_propagate(int64_t n_orb, const double *onsite, int64_t n_hop, const int32_t *hop_i, const int32_t *hop_j,
                     const double *hop_val, int hops_full, const double *psi_start, const double *psi0, int n_step,
                     double dt, double rescale, double tol, double *corr, double *norm2, double *psi_final)
{
    if (n_orb < 0 || n_step < 0 || !(rescale > 0.0) || !(dt >= 0.0)) return ORACLE_EINVAL;
    enum { KCAP = 4096 };
    int K = 0;
    double *coeff = (double *)malloc(sizeof(double) * 2 * KCAP);
    if (!coeff) return ORACLE_ENOMEM;
    int rc = oracle_cheb_coeff(rescale * dt, tol, KCAP, &K, coeff);
    if (rc) { free(coeff); return rc; }
    size_t vb = sizeof(double) * 2 * (size_t)(n_orb > 0 ? n_orb : 1);
    double *buf0 = (double *)malloc(vb), *buf1 = (double *)malloc(vb), *wf_out = (double *)malloc(vb), *psi = (double *)malloc(vb);
    if (!buf0 || !buf1 || !wf_out || !psi) { free(coeff); free(buf0); free(buf1); free(wf_out); free(psi); return ORACLE_ENOMEM; }
    memcpy(psi, psi_start, sizeof(double) * 2 * (size_t)n_orb);
    const double s = rescale;
    for (int n = 0; n < n_step; ++n) {
        double *p0 = buf0, *p1 = buf1, *p2;
        memcpy(p0, psi, sizeof(double) * 2 * (size_t)n_orb);                       /* T_0 = psi            */
        memset(wf_out, 0, sizeof(double) * 2 * (size_t)n_orb);
        axpy_c(n_orb, coeff[0], coeff[1], p0, wf_out);                             /* wf_out = c_0 T_0     */
        if (K > 1) {
            amxsy_hops(n_orb, onsite, n_hop, hop_i, hop_j, hop_val, hops_full, 1.0 / s, p0, p1, 0); /* T_1 = H' T_0 */
            axpy_c(n_orb, coeff[2], coeff[3], p1, wf_out);                         /* += c_1 T_1           */
        }
        for (int k = 2; k < K; ++k) {
            p2 = p0;
            amxsy_hops(n_orb, onsite, n_hop, hop_i, hop_j, hop_val, hops_full, 2.0 / s, p1, p0, 1);
            axpy_c(n_orb, coeff[2 * k], coeff[2 * k + 1], p2, wf_out);
            p0 = p1;
            p1 = p2;
        }
        memcpy(psi, wf_out, sizeof(double) * 2 * (size_t)n_orb);
        double cr, ci, nn;
        dots(n_orb, psi0, psi, &cr, &ci, &nn);
        corr[2 * n] = cr; corr[2 * n + 1] = ci;
        if (norm2) norm2[n] = nn;
    }
    if (psi_final) memcpy(psi_final, psi, sizeof(double) * 2 * (size_t)n_orb);
    free(coeff); free(buf0); free(buf1); free(wf_out); free(psi);
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------------------
 * Row form on the canonical CSR with OpenMP over rows ("for each initial state, the propagation is
 * parallelized using OpenMP threads").  Same loop, same order of terms; only the H application
 * is gathered by row instead of scattered by hop.  Checked against oracle_propagate in the pins; used for the
 * timed cpu_baseline and for prefix/windowed parity at the large configs.
 * ------------------------------------------------------------------------------------------------------- */
int oracle_propagate_csr(int64_t n_orb, const int64_t *rowptr, const int32_t *col, const double *val,
                         const double *psi_start, const double *psi0, int n_step, double dt, double rescale, double tol,
                         double *corr, double *norm2, double *psi_final)
{
    if (n_orb < 0 || n_step < 0 || !(rescale > 0.0) || !(dt >= 0.0)) return ORACLE_EINVAL;
    enum { KCAP = 4096 };
    int K = 0;
    double *coeff = (double *)malloc(sizeof(double) * 2 * KCAP);
    if (!coeff) return ORACLE_ENOMEM;
    int rc = oracle_cheb_coeff(rescale * dt, tol, KCAP, &K, coeff);
    if (rc) { free(coeff); return rc; }
    size_t vb = sizeof(double) * 2 * (size_t)(n_orb > 0 ? n_orb : 1);
    double *buf0 = (double *)malloc(vb), *buf1 = (double *)malloc(vb), *wf_out = (double *)malloc(vb), *psi = (double *)malloc(vb);
    if (!buf0 || !buf1 || !wf_out || !psi) { free(coeff); free(buf0); free(buf1); free(wf_out); free(psi); return ORACLE_ENOMEM; }
    memcpy(psi, psi_start, sizeof(double) * 2 * (size_t)n_orb);
    const double s = rescale;
    for (int n = 0; n < n_step; ++n) {
        double *p0 = buf0, *p1 = buf1, *p2;
        const double c0r = coeff[0], c0i = coeff[1];
        const double c1r = K > 1 ? coeff[2] : 0.0, c1i = K > 1 ? coeff[3] : 0.0;
        const double a1 = 1.0 / s;
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < n_orb; ++i) {                                      /* T_0, T_1, first two terms */
            double xr = psi[2 * i], xi = psi[2 * i + 1];
            p0[2 * i] = xr; p0[2 * i + 1] = xi;
            double hr = 0.0, hi = 0.0;
            if (K > 1) {
                for (int64_t p = rowptr[i]; p < rowptr[i + 1]; ++p) {
                    double vr = a1 * val[2 * p], vi = a1 * val[2 * p + 1];
                    int64_t j = col[p];
                    hr += vr * psi[2 * j] - vi * psi[2 * j + 1];
                    hi += vr * psi[2 * j + 1] + vi * psi[2 * j];
                }
            }
            p1[2 * i] = hr; p1[2 * i + 1] = hi;
            wf_out[2 * i]     = (c0r * xr - c0i * xi) + (c1r * hr - c1i * hi);
            wf_out[2 * i + 1] = (c0r * xi + c0i * xr) + (c1r * hi + c1i * hr);
        }
        for (int k = 2; k < K; ++k) {
            p2 = p0;
            const double a = 2.0 / s, cr = coeff[2 * k], ci = coeff[2 * k + 1];
#pragma omp parallel for schedule(static)
            for (int64_t i = 0; i < n_orb; ++i) {                                  /* amxsy + axpy, row i */
                double hr = -p0[2 * i], hi = -p0[2 * i + 1];
                for (int64_t p = rowptr[i]; p < rowptr[i + 1]; ++p) {
                    double vr = a * val[2 * p], vi = a * val[2 * p + 1];
                    int64_t j = col[p];
                    hr += vr * p1[2 * j] - vi * p1[2 * j + 1];
                    hi += vr * p1[2 * j + 1] + vi * p1[2 * j];
                }
                p0[2 * i] = hr; p0[2 * i + 1] = hi;
                wf_out[2 * i]     += cr * hr - ci * hi;
                wf_out[2 * i + 1] += cr * hi + ci * hr;
            }
            p0 = p1;
            p1 = p2;
        }
        long double sr = 0.0L, si = 0.0L, nn = 0.0L;
#pragma omp parallel for schedule(static) reduction(+ : sr, si, nn)
        for (int64_t i = 0; i < n_orb; ++i) {
            double br = wf_out[2 * i], bi = wf_out[2 * i + 1];
            psi[2 * i] = br; psi[2 * i + 1] = bi;
            long double ar = psi0[2 * i], ai = psi0[2 * i + 1];
            sr += ar * (long double)br + ai * (long double)bi;
            si += ar * (long double)bi - ai * (long double)br;
            nn += (long double)br * br + (long double)bi * bi;
        }
        corr[2 * n] = (double)sr; corr[2 * n + 1] = (double)si;
        if (norm2) norm2[n] = (double)nn;
    }
    if (psi_final) memcpy(psi_final, psi, sizeof(double) * 2 * (size_t)n_orb);
    free(coeff); free(buf0); free(buf1); free(wf_out); free(psi);
    return ORACLE_OK;
}

/* y = H x from the hop list (no scaling) -- exposed so that the pins can compare it with a dense matrix. */
int oracle_apply_h(int64_t n_orb, const double *onsite, int64_t n_hop, const int32_t *hop_i, const int32_t *hop_j,
                   const double *hop_val, int hops_full, const double *x, double *y)
{
    if (n_orb < 0 || n_hop < 0) return ORACLE_EINVAL;
    amxsy_hops(n_orb, onsite, n_hop, hop_i, hop_j, hop_val, hops_full, 1.0, x, y, 0);
    return ORACLE_OK;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

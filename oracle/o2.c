/* Oracle tier O2 -- TEST INFRASTRUCTURE, not the product (see oracle/__init__.py).
 *
 * Plain C99 + OpenMP, float64.  Shares no code with the CUDA path.
 *
 * What it computes ("plain definition", steps 1-6), for every walker w
 * against the trial  |Psi_T> = sum_I c_I |D_I>  (Eq. 15, orthogonal CI expansion):
 *
 *   for every determinant I and spin s, with occ_I the ASCENDING occupation list:
 *     O_I  = psi[occ_I, :]                      (n x n)      Psi_T^+ phi of Eq. 13
 *     d_I  = det O_I                                         Eq. 13
 *     Th_I = psi O_I^-1                         (N x n)      Eq. 14: G_I[occ_I[l], q] = Th_I[q, l]
 *   ovlp = sum_I c_I d_I^a d_I^b                             Eq. 15 + Eq. 13
 *   G^s  = sum_I c_I d_I^a d_I^b G_I^s / ovlp                mixed Green's function
 *   fb_g = sum_pq L^g_pq (G^a + G^b)_pq                      Eq. 7 without the factor -sqrt(dtau)
 *   E_I  = sum_pq h_pq (G_I^a+G_I^b)_pq
 *          + 1/2 sum_g [ X_g^2 - sum_s sum_pqrs L^g_pq L^g_rs G^s_I,ps G^s_I,rq ]     Eq. 2
 *   E    = e0 + sum_I c_I d_I^a d_I^b E_I / ovlp
 *
 * "Touching only non-zero rows": G_I has n non-zero rows, so with (L^g psi) computed once per walker
 *     T_I^g = (L^g psi)[occ_I, :] O_I^-1  (n x n),   X_g = sum_s tr T_I^{g,s},
 *     sum_pqrs L_pq L_rs G_ps G_rq = tr(T_I^g T_I^g),   sum_pq h_pq G_pq = tr((h psi)[occ_I,:] O_I^-1).
 * That is the same arithmetic as tier O1 (oracle/msd_oracle.py) with the zero rows skipped; the two are
 * compared in tests/test_oracle_pins.py.  One LU + inverse per (walker, determinant, spin): no Wick's theorem,
 * no reuse between determinants (the "naive approach").
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <tgmath.h>   /* cabs / creal / cimag follow the type of REAL */
#ifdef _OPENMP
#include <omp.h>
#endif

/* REAL is the working precision: double (the oracle), or long double when built with -DREAL="long double" for the
 * noise-floor pin P12: same statements, wider type.  The interface stays float64 either way. */
#ifndef REAL
#define REAL double
#endif
typedef REAL real;
typedef REAL complex cplx;
typedef double complex dcplx;

/* LU with partial pivoting of the n x n matrix a (row-major, overwritten); returns det, writes the inverse
 * to inv (row-major).  Returns 0 and leaves inv undefined if a pivot is exactly zero. */
static cplx lu_det_inverse(int n, cplx *a, cplx *inv, int *piv)
{
    cplx det = 1.0;
    for (int i = 0; i < n; i++) piv[i] = i;
    for (int j = 0; j < n; j++) {
        int p = j;
        real best = cabs(a[j * n + j]);
        for (int i = j + 1; i < n; i++) {
            real v = cabs(a[i * n + j]);
            if (v > best) { best = v; p = i; }
        }
        if (best == 0.0) return 0.0;
        if (p != j) {
            for (int c = 0; c < n; c++) { cplx t = a[j * n + c]; a[j * n + c] = a[p * n + c]; a[p * n + c] = t; }
            int t = piv[j]; piv[j] = piv[p]; piv[p] = t;
            det = -det;
        }
        det *= a[j * n + j];
        cplx r = 1.0 / a[j * n + j];
        for (int i = j + 1; i < n; i++) {
            cplx l = a[i * n + j] * r;
            a[i * n + j] = l;
            for (int c = j + 1; c < n; c++) a[i * n + c] -= l * a[j * n + c];
        }
    }
    /* solve A X = I column by column:  P A = L U  =>  X[:,c] = U^-1 L^-1 P e_c */
    for (int c = 0; c < n; c++) {
        cplx y[64];
        for (int i = 0; i < n; i++) {
            cplx s = (piv[i] == c) ? 1.0 : 0.0;
            for (int k = 0; k < i; k++) s -= a[i * n + k] * y[k];
            y[i] = s;
        }
        for (int i = n - 1; i >= 0; i--) {
            cplx s = y[i];
            for (int k = i + 1; k < n; k++) s -= a[i * n + k] * inv[k * n + c];
            inv[i * n + c] = s / a[i * n + i];
        }
    }
    return det;
}

/* per-spin, per-determinant work.  Returns d_I; fills tr_h = tr((h psi)[occ,:] O^-1), X[g] += tr T^g,
 * ex[g] += tr(T^g T^g); if Gacc != NULL accumulates wgt * G_I is done by the caller via theta. */
typedef struct {
    int N, n, ng;
    const cplx *psi;   /* [N][n] */
    const cplx *hpsi;  /* [N][n] = h1 psi */
    const cplx *Lpsi;  /* [ng][N][n] = L^g psi */
} spin_ctx;

static cplx det_terms(const spin_ctx *s, const int *occ, int want_energy, int want_theta,
                      cplx *O, cplx *Oinv, int *piv, cplx *theta /* [N][n] */,
                      cplx *tr_h, cplx *X /* [ng] += */, cplx *ex /* [ng] += */,
                      real *Tr, real *Ti, real *Ir, real *Ii)
{
    const int n = s->n, N = s->N, ng = s->ng;
    if (n == 0) { *tr_h = 0.0; return 1.0; }
    for (int l = 0; l < n; l++)
        for (int i = 0; i < n; i++) O[l * n + i] = s->psi[(size_t)occ[l] * n + i];
    cplx d = lu_det_inverse(n, O, Oinv, piv);
    if (d == 0.0) { *tr_h = 0.0; return 0.0; }   /* contributes nothing to any numerator (all carry d_I) */
    if (want_theta) {
        for (int q = 0; q < N; q++)
            for (int l = 0; l < n; l++) {
                cplx acc = 0.0;
                for (int m = 0; m < n; m++) acc += s->psi[(size_t)q * n + m] * Oinv[m * n + l];
                theta[(size_t)q * n + l] = acc;
            }
    }
    if (!want_energy) return d;
    /* tr((h psi)[occ,:] O^-1) */
    cplx th = 0.0;
    for (int l = 0; l < n; l++)
        for (int m = 0; m < n; m++) th += s->hpsi[(size_t)occ[l] * n + m] * Oinv[m * n + l];
    *tr_h = th;
    /* split O^-1 once for the inner loops */
    for (int k = 0; k < n * n; k++) { Ir[k] = creal(Oinv[k]); Ii[k] = cimag(Oinv[k]); }
    for (int g = 0; g < ng; g++) {
        const cplx *Lp = s->Lpsi + (size_t)g * N * n;
        /* T = (L^g psi)[occ,:] O^-1 */
        for (int l = 0; l < n; l++) {
            real *tr = Tr + l * n, *ti = Ti + l * n;
            for (int i = 0; i < n; i++) { tr[i] = 0.0; ti[i] = 0.0; }
            const cplx *row = Lp + (size_t)occ[l] * n;
            for (int m = 0; m < n; m++) {
                const real ar = creal(row[m]), ai = cimag(row[m]);
                const real *br = Ir + m * n, *bi = Ii + m * n;
                for (int i = 0; i < n; i++) {
                    tr[i] += ar * br[i] - ai * bi[i];
                    ti[i] += ar * bi[i] + ai * br[i];
                }
            }
        }
        real xr = 0.0, xi = 0.0, er = 0.0, ei = 0.0;
        for (int l = 0; l < n; l++) { xr += Tr[l * n + l]; xi += Ti[l * n + l]; }
        for (int l = 0; l < n; l++)
            for (int i = 0; i < n; i++) {
                const real ar = Tr[l * n + i], ai = Ti[l * n + i], br = Tr[i * n + l], bi = Ti[i * n + l];
                er += ar * br - ai * bi;
                ei += ar * bi + ai * br;
            }
        X[g] += xr + I * xi;
        ex[g] += er + I * ei;
    }
    return d;
}

/* want: bit 0 overlap (always), bit 1 Green's function + force bias, bit 2 energy.
 * Layouts (all row-major, C order): h1[N][N], L[ng][N][N], occa[nd][na], occb[nd][nb], ci[nd],
 * phi_a[nw][N][na], phi_b[nw][N][nb] complex128; outputs ovlp[nw], G[nw][2][N][N] (may be NULL),
 * fb[nw][ng], E[nw][3] = (E, E1, E2).  kappa[nw] (may be NULL) = sum_I |c_I d_I^a d_I^b| / |ovlp|.
 * Returns 0, or -1 on bad arguments / allocation failure. */
int msd_oracle_o2(int N, int na, int nb, int ng, long nd, int nw,
                  const double *h1, const double *L, double e0,
                  const int *occa, const int *occb, const double *ci,
                  const dcplx *phi_a, const dcplx *phi_b, int want,
                  dcplx *ovlp, dcplx *G, dcplx *fb, dcplx *E, double *kappa, int nthreads)
{
    if (N <= 0 || na < 0 || nb < 0 || na > 64 || nb > 64 || nd <= 0 || nw < 0) return -1;
    const int want_g = (want & 2) != 0, want_e = (want & 4) != 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
    int nt = omp_get_max_threads();
#else
    int nt = 1;
#endif
    const int nmax = na > nb ? na : nb;
    cplx *hpsi[2], *Lpsi[2], *psiw[2];
    const int ns[2] = {na, nb};
    for (int s = 0; s < 2; s++) {
        hpsi[s] = (cplx *)malloc(sizeof(cplx) * (size_t)N * (ns[s] + 1));
        Lpsi[s] = (cplx *)malloc(sizeof(cplx) * (size_t)(want_e ? ng : 1) * N * (ns[s] + 1));
        psiw[s] = (cplx *)malloc(sizeof(cplx) * (size_t)N * (ns[s] + 1));   /* the walker in the working precision */
        if (!hpsi[s] || !Lpsi[s] || !psiw[s]) return -1;
    }
    /* per-determinant numerators, summed sequentially afterwards (thread-count independent) */
    cplx *wI = (cplx *)malloc(sizeof(cplx) * nd);
    cplx *e1I = (cplx *)malloc(sizeof(cplx) * nd);
    cplx *e2I = (cplx *)malloc(sizeof(cplx) * nd);
    cplx *Gthr = want_g ? (cplx *)calloc((size_t)nt * 2 * N * N, sizeof(cplx)) : NULL;
    if (!wI || !e1I || !e2I || (want_g && !Gthr)) return -1;

    for (int w = 0; w < nw; w++) {
        const dcplx *psi_in[2] = {phi_a + (size_t)w * N * na, phi_b + (size_t)w * N * nb};
        for (int s = 0; s < 2; s++)
            for (size_t k = 0; k < (size_t)N * ns[s]; k++) psiw[s][k] = psi_in[s][k];
        const cplx *psi[2] = {psiw[0], psiw[1]};
        for (int s = 0; s < 2; s++) {
            const int n = ns[s];
            if (!want_e) continue;
            for (int p = 0; p < N; p++)
                for (int i = 0; i < n; i++) {
                    cplx acc = 0.0;
                    for (int q = 0; q < N; q++) acc += h1[(size_t)p * N + q] * psi[s][(size_t)q * n + i];
                    hpsi[s][(size_t)p * n + i] = acc;
                }
#pragma omp parallel for schedule(static)
            for (int g = 0; g < ng; g++)
                for (int p = 0; p < N; p++)
                    for (int i = 0; i < n; i++) {
                        cplx acc = 0.0;
                        const double *Lrow = L + ((size_t)g * N + p) * N;
                        for (int q = 0; q < N; q++) acc += Lrow[q] * psi[s][(size_t)q * n + i];
                        Lpsi[s][((size_t)g * N + p) * n + i] = acc;
                    }
        }
        if (want_g) memset(Gthr, 0, sizeof(cplx) * (size_t)nt * 2 * N * N);
#pragma omp parallel
        {
#ifdef _OPENMP
            const int tid = omp_get_thread_num();
#else
            const int tid = 0;
#endif
            cplx *O = (cplx *)malloc(sizeof(cplx) * (nmax * nmax + 1));
            cplx *Oinv = (cplx *)malloc(sizeof(cplx) * (nmax * nmax + 1));
            cplx *theta = (cplx *)malloc(sizeof(cplx) * ((size_t)N * nmax + 1));
            cplx *X = (cplx *)malloc(sizeof(cplx) * (ng + 1));
            cplx *ex = (cplx *)malloc(sizeof(cplx) * (ng + 1));
            real *Tr = (real *)malloc(sizeof(real) * 4 * (nmax * nmax + 1));
            real *Ti = Tr + (nmax * nmax + 1), *Ir = Ti + (nmax * nmax + 1), *Ii = Ir + (nmax * nmax + 1);
            int piv[64];
#pragma omp for schedule(dynamic, 16)
            for (long Id = 0; Id < nd; Id++) {
                cplx d[2], trh[2];
                if (want_e) for (int g = 0; g < ng; g++) { X[g] = 0.0; ex[g] = 0.0; }
                /* both determinants first: the weight c_I d_a d_b multiplies each spin's G_I */
                spin_ctx sc[2];
                const int *occ[2] = {occa + (size_t)Id * na, occb + (size_t)Id * nb};
                for (int s = 0; s < 2; s++) {
                    sc[s].N = N; sc[s].n = ns[s]; sc[s].ng = ng;
                    sc[s].psi = psi[s]; sc[s].hpsi = hpsi[s]; sc[s].Lpsi = Lpsi[s];
                }
                /* pass 1: determinants (and energy traces) */
                for (int s = 0; s < 2; s++)
                    d[s] = det_terms(&sc[s], occ[s], want_e, 0, O, Oinv, piv, theta, &trh[s], X, ex, Tr, Ti, Ir, Ii);
                const cplx wgt = ci[Id] * d[0] * d[1];
                wI[Id] = wgt;
                e1I[Id] = 0.0; e2I[Id] = 0.0;
                if (wgt == 0.0) continue;
                if (want_e) {
                    cplx e2 = 0.0;
                    for (int g = 0; g < ng; g++) e2 += X[g] * X[g] - ex[g];
                    e1I[Id] = wgt * (trh[0] + trh[1]);
                    e2I[Id] = wgt * 0.5 * e2;
                }
                if (want_g) {
                    /* pass 2: Theta_I per spin, accumulate wgt * G_I:  G_I[occ[l], q] = Theta_I[q, l] */
                    for (int s = 0; s < 2; s++) {
                        cplx dummy;
                        det_terms(&sc[s], occ[s], 0, 1, O, Oinv, piv, theta, &dummy, X, ex, Tr, Ti, Ir, Ii);
                        cplx *Gs = Gthr + ((size_t)tid * 2 + s) * N * N;
                        const int n = ns[s];
                        for (int l = 0; l < n; l++)
                            for (int q = 0; q < N; q++) Gs[(size_t)occ[s][l] * N + q] += wgt * theta[(size_t)q * n + l];
                    }
                }
            }
            free(O); free(Oinv); free(theta); free(X); free(ex); free(Tr);
        }
        cplx den = 0.0, n1 = 0.0, n2 = 0.0;
        real sabs = 0.0;
        for (long Id = 0; Id < nd; Id++) { den += wI[Id]; n1 += e1I[Id]; n2 += e2I[Id]; sabs += cabs(wI[Id]); }
        ovlp[w] = den;
        if (kappa) kappa[w] = sabs / cabs(den);
        if (want_e) {
            E[(size_t)w * 3 + 1] = n1 / den;
            E[(size_t)w * 3 + 2] = n2 / den;
            E[(size_t)w * 3 + 0] = e0 + n1 / den + n2 / den;
        }
        if (want_g) {
            cplx *Gw = Gthr; /* reduce the thread copies into copy 0, in thread order */
            for (int t = 1; t < nt; t++)
                for (size_t k = 0; k < (size_t)2 * N * N; k++) Gw[k] += Gthr[(size_t)t * 2 * N * N + k];
            for (size_t k = 0; k < (size_t)2 * N * N; k++) Gw[k] /= den;
            if (G) for (size_t k = 0; k < (size_t)2 * N * N; k++) G[(size_t)w * 2 * N * N + k] = Gw[k];
            for (int g = 0; g < ng; g++) {
                cplx acc = 0.0;
                const double *Lg = L + (size_t)g * N * N;
                for (size_t k = 0; k < (size_t)N * N; k++) acc += Lg[k] * (Gw[k] + Gw[(size_t)N * N + k]);
                fb[(size_t)w * ng + g] = acc;
            }
        }
    }
    for (int s = 0; s < 2; s++) { free(hpsi[s]); free(Lpsi[s]); free(psiw[s]); }
    free(wI); free(e1I); free(e2I); free(Gthr);
    return 0;
}

int msd_oracle_o2_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

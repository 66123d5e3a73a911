/* CPU restatement of the generalized-Wick's-theorem algorithm W1-W10,
 * multi-threaded with OpenMP: the like-for-like CPU baseline of SURVEY.md 8(f) f1 (the paper's own comparison is
 * Wick-on-CPU vs Wick-on-GPU).
 *
 * TEST / BENCH INFRASTRUCTURE (see oracle/__init__.py): nothing under paper_2406_08314_b200/ uses it, and it shares no
 * code with the CUDA path.  It is NOT the parity oracle (that is O0/O1/O2, which never use Wick's theorem); it is checked
 * against O2 in tests/test_oracle_pins.py and timed by bench.py as "cpu_wick_baseline".
 * Limitation (by design, it is a baseline): cofactors are taken as R * M^-1 at every level >= 3, so exactly singular
 * minors (walker == reference determinant) are not supported.
 *
 * Per walker and spin (Eq. 13-15 through the matrix-determinant lemma):
 *   W1  O0 = psi[occ0,:], det0, Theta = psi O0^-1, g[h,p] = Theta[p, pos(h)]
 *   W2  M[a,b] = g[h_a,p_b], R = det M            W3  W = sum c~ R^a R^b, ovlp = det0^a det0^b W
 *   W4  A = R M^-1,  C^s[p_b,h_a] += c~ R^sbar A[b,a]
 *   W6  fb_g = sum_s [ X0^s_g + (1/W) sum_x C^s[x] B^{s,g}[x] ]
 *   W7  T^g = (L^g Theta)[occ0 rows], X0_g = tr T^g, Ex0_g = tr T^g T^g, B^g = (L^g Theta)[virt] - Theta[virt] T^g
 *   W8  E1 = sum_s tr T^{h1,s} + (1/W) sum C.Hrot
 *   W9  E2 = 1/2 sum_g [(X0^a+X0^b)^2 - Ex0^a - Ex0^b] + (1/W) [ sum C.F + E2nd ],  V^{ss'} = sum_g B^{s,g} (x) B^{s',g}
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cd;
#define KMAX 16

int msd_wick_cpu_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* in-place inverse by Gauss-Jordan with partial pivoting; returns det (0 if singular: a is then garbage) */
static cd inv_det(cd* a, int n)
{
    int piv[64];
    cd det = 1.0;
    for (int j = 0; j < n; j++) {
        int p = j; double best = cabs(a[j * n + j]);
        for (int i = j + 1; i < n; i++) { double v = cabs(a[i * n + j]); if (v > best) { best = v; p = i; } }
        piv[j] = p;
        if (best == 0.0) return 0.0;
        if (p != j) { for (int c = 0; c < n; c++) { cd t = a[j * n + c]; a[j * n + c] = a[p * n + c]; a[p * n + c] = t; } det = -det; }
        cd pv = a[j * n + j]; det *= pv;
        cd r = 1.0 / pv;
        a[j * n + j] = 1.0;
        for (int c = 0; c < n; c++) a[j * n + c] *= r;
        for (int i = 0; i < n; i++) {
            if (i == j) continue;
            cd f = a[i * n + j]; a[i * n + j] = 0.0;
            for (int c = 0; c < n; c++) a[i * n + c] -= f * a[j * n + c];
        }
    }
    for (int j = n - 1; j >= 0; j--)
        if (piv[j] != j) for (int i = 0; i < n; i++) { cd t = a[i * n + j]; a[i * n + j] = a[i * n + piv[j]]; a[i * n + piv[j]] = t; }
    return det;
}

typedef struct {
    int n, no, nv, P;
    const int* occ0;
    int act_o[64], act_v[256], pos_o[64];   /* orbital of active hole h / virtual r; position of act_o[h] in occ0 */
    int loc_o[1024], loc_v[1024];            /* orbital -> window-local index (or -1) */
} Spin;

/* active window (reading A10) and in-place -> sorted parity of every determinant of one spin */
static int spin_setup(Spin* s, int N, int n, const int* occ0, int64_t nd, const int64_t* off, const int* holes, const int* parts,
                      signed char* phase)
{
    if (N > 1024 || n > 64) return -1;
    s->n = n; s->occ0 = occ0;
    for (int q = 0; q < N; q++) { s->loc_o[q] = -1; s->loc_v[q] = -1; }
    for (int64_t e = 0; e < off[nd]; e++) { s->loc_o[holes[e]] = 0; s->loc_v[parts[e]] = 0; }
    s->no = s->nv = 0;
    for (int q = 0; q < N; q++) {
        if (s->loc_o[q] == 0) { if (s->no >= 64) return -1; s->act_o[s->no] = q; s->loc_o[q] = s->no++; }
        if (s->loc_v[q] == 0) { if (s->nv >= 256) return -1; s->act_v[s->nv] = q; s->loc_v[q] = s->nv++; }
    }
    for (int h = 0; h < s->no; h++) {
        s->pos_o[h] = -1;
        for (int l = 0; l < n; l++) if (occ0[l] == s->act_o[h]) s->pos_o[h] = l;
        if (s->pos_o[h] < 0) return -2;
    }
    s->P = s->no * s->nv;
#pragma omp parallel for schedule(static)
    for (int64_t d = 0; d < nd; d++) {
        int list[64];
        for (int l = 0; l < n; l++) list[l] = occ0[l];
        int k = (int)(off[d + 1] - off[d]);
        int hs[KMAX], ps[KMAX];
        for (int a = 0; a < k; a++) { hs[a] = holes[off[d] + a]; ps[a] = parts[off[d] + a]; }
        for (int a = 1; a < k; a++) {         /* a-th smallest hole <-> a-th smallest particle (reading A7) */
            int v = hs[a], j = a; while (j > 0 && hs[j - 1] > v) { hs[j] = hs[j - 1]; j--; } hs[j] = v;
            v = ps[a]; j = a; while (j > 0 && ps[j - 1] > v) { ps[j] = ps[j - 1]; j--; } ps[j] = v;
        }
        for (int a = 0; a < k; a++)
            for (int l = 0; l < n; l++) if (occ0[l] == hs[a]) list[l] = ps[a];
        int inv = 0;
        for (int i = 0; i < n; i++) for (int j = i + 1; j < n; j++) inv += list[i] > list[j];
        phase[d] = (inv & 1) ? -1 : 1;
    }
    return 0;
}

typedef struct {           /* per-walker, per-spin intermediates */
    cd det0;
    cd* theta;             /* [N][n] */
    cd* g;                 /* [P], x = p*no + h */
    cd* B;                 /* [ng+1][P]  (slice ng = h1 -> Hrot) */
    cd* X0;                /* [ng] */
    cd* FK;                /* [P]  sum_g (Bfull T)[r][pos_o[h]] */
    cd* F;                 /* [P] */
    cd ex0, e1_0;
} WS;

/* W1 */
static int reference(const Spin* s, int N, const cd* psi, WS* w)
{
    const int n = s->n;
    w->det0 = 1.0;
    if (n == 0) return 0;
    cd* O = (cd*)malloc(sizeof(cd) * n * n);
    for (int l = 0; l < n; l++) for (int i = 0; i < n; i++) O[l * n + i] = psi[(size_t)s->occ0[l] * n + i];
    w->det0 = inv_det(O, n);
    if (w->det0 == 0.0) { free(O); return 1; }
#pragma omp parallel for schedule(static)
    for (int q = 0; q < N; q++)
        for (int i = 0; i < n; i++) {
            cd t = 0.0;
            for (int l = 0; l < n; l++) t += psi[(size_t)q * n + l] * O[l * n + i];
            w->theta[(size_t)q * n + i] = t;
        }
    for (int p = 0; p < s->nv; p++)
        for (int h = 0; h < s->no; h++) w->g[p * s->no + h] = w->theta[(size_t)s->act_v[p] * n + s->pos_o[h]];
    free(O);
    return 0;
}

/* W7 for one spin: slices g = 0..ng-1 are L^g, slice ng is h1 */
static void half_rotate(const Spin* s, int N, int ng, const double* h1, const double* L, WS* w)
{
    const int n = s->n, no = s->no, nv = s->nv, P = s->P;
    w->ex0 = 0.0; w->e1_0 = 0.0;
    for (int x = 0; x < P; x++) w->FK[x] = 0.0;
    if (n == 0) { for (int g = 0; g < ng; g++) w->X0[g] = 0.0; return; }
    double exr = 0.0, exi = 0.0;
#pragma omp parallel
    {
        cd* T = (cd*)malloc(sizeof(cd) * (n * n + (size_t)nv * n * 2));
        cd* Lv = T + n * n;
        cd* Bf = Lv + (size_t)nv * n;
        cd* fk = (cd*)calloc(P > 0 ? P : 1, sizeof(cd));
        double lexr = 0.0, lexi = 0.0;
#pragma omp for schedule(static)
        for (int g = 0; g <= ng; g++) {
            const double* Lg = (g < ng) ? L + (size_t)g * N * N : h1;
            for (int l = 0; l < n; l++)
                for (int i = 0; i < n; i++) {
                    cd t = 0.0;
                    const double* row = Lg + (size_t)s->occ0[l] * N;
                    for (int q = 0; q < N; q++) t += row[q] * w->theta[(size_t)q * n + i];
                    T[l * n + i] = t;
                }
            for (int r = 0; r < nv; r++)
                for (int i = 0; i < n; i++) {
                    cd t = 0.0;
                    const double* row = Lg + (size_t)s->act_v[r] * N;
                    for (int q = 0; q < N; q++) t += row[q] * w->theta[(size_t)q * n + i];
                    Lv[r * n + i] = t;
                }
            cd tr = 0.0;
            for (int l = 0; l < n; l++) tr += T[l * n + l];
            for (int r = 0; r < nv; r++)
                for (int i = 0; i < n; i++) {
                    cd t = Lv[r * n + i];
                    const cd* th = w->theta + (size_t)s->act_v[r] * n;
                    for (int l = 0; l < n; l++) t -= th[l] * T[l * n + i];
                    Bf[r * n + i] = t;
                }
            for (int r = 0; r < nv; r++)
                for (int h = 0; h < no; h++) w->B[(size_t)g * P + r * no + h] = Bf[r * n + s->pos_o[h]];
            if (g < ng) {
                w->X0[g] = tr;
                cd ex = 0.0;
                for (int l = 0; l < n; l++) for (int i = 0; i < n; i++) ex += T[l * n + i] * T[i * n + l];
                lexr += creal(ex); lexi += cimag(ex);
                for (int r = 0; r < nv; r++)
                    for (int h = 0; h < no; h++) {
                        cd t = 0.0;
                        for (int i = 0; i < n; i++) t += Bf[r * n + i] * T[i * n + s->pos_o[h]];
                        fk[r * no + h] += t;
                    }
            } else {
                w->e1_0 = tr;
            }
        }
#pragma omp critical
        {
            exr += lexr; exi += lexi;
            for (int x = 0; x < P; x++) w->FK[x] += fk[x];
        }
        free(T); free(fk);
    }
    w->ex0 = exr + exi * I;
}

/* V[x][y] = sum_g Bs[g][x] Bt[g][y] */
static void vtensor(int ng, int Ps, int Pt, const cd* Bs, const cd* Bt, cd* V)
{
#pragma omp parallel for schedule(static)
    for (int x = 0; x < Ps; x++)
        for (int y = 0; y < Pt; y++) {
            cd t = 0.0;
            for (int g = 0; g < ng; g++) t += Bs[(size_t)g * Ps + x] * Bt[(size_t)g * Pt + y];
            V[(size_t)x * Pt + y] = t;
        }
}

/* one spin of one determinant: pair indices x[a*k+b] = (p_b, h_a), R = det M, A[b*k+a] = R (M^-1)[b][a] */
static cd spin_det(const Spin* s, int k, const int* holes, const int* parts, const cd* g, int* x, cd* A)
{
    if (k == 0) return 1.0;
    int h[KMAX], p[KMAX];
    for (int a = 0; a < k; a++) { h[a] = s->loc_o[holes[a]]; p[a] = s->loc_v[parts[a]]; }
    for (int a = 1; a < k; a++) {             /* ascending, a-th hole with a-th particle (reading A7) */
        int v = h[a], j = a; while (j > 0 && h[j - 1] > v) { h[j] = h[j - 1]; j--; } h[j] = v;
        v = p[a]; j = a; while (j > 0 && p[j - 1] > v) { p[j] = p[j - 1]; j--; } p[j] = v;
    }
    cd M[KMAX * KMAX];
    for (int a = 0; a < k; a++)
        for (int b = 0; b < k; b++) { x[a * k + b] = p[b] * s->no + h[a]; M[a * k + b] = g[x[a * k + b]]; }
    if (k == 1) { A[0] = 1.0; return M[0]; }
    if (k == 2) {
        A[0] = M[3]; A[1] = -M[1]; A[2] = -M[2]; A[3] = M[0];     /* adj: A[b*2+a] = cofactor of M[a][b] */
        return M[0] * M[3] - M[1] * M[2];
    }
    cd R = inv_det(M, k);
    for (int e = 0; e < k * k; e++) A[e] = (R == 0.0) ? 0.0 : R * M[e];
    return R;
}

/* bits: 1 overlap, 2 force bias, 4 energy.  Walkers are processed one after another; all threads work inside a walker
 * (dense steps over Cholesky slices, the determinant loop over determinants with per-thread accumulators). */
int msd_wick_cpu(int N, int na, int nb, int ng, int64_t nd, int nw, const double* h1, const double* L, double e0,
                 const int* occ_ref_a, const int* occ_ref_b, const int64_t* off_a, const int* holes_a, const int* parts_a,
                 const int64_t* off_b, const int* holes_b, const int* parts_b, const double* ci, const cd* phi_a,
                 const cd* phi_b, int bits, cd* ovlp, cd* fb, cd* E, int nthreads)
{
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
    Spin* sp = (Spin*)malloc(2 * sizeof(Spin));
    signed char* ph[2] = {(signed char*)malloc(nd > 0 ? nd : 1), (signed char*)malloc(nd > 0 ? nd : 1)};
    int rc = spin_setup(&sp[0], N, na, occ_ref_a, nd, off_a, holes_a, parts_a, ph[0]);
    if (!rc) rc = spin_setup(&sp[1], N, nb, occ_ref_b, nd, off_b, holes_b, parts_b, ph[1]);
    if (rc) { free(sp); free(ph[0]); free(ph[1]); return rc; }
    for (int64_t d = 0; d < nd; d++)
        if (off_a[d + 1] - off_a[d] > KMAX || off_b[d + 1] - off_b[d] > KMAX) { free(sp); free(ph[0]); free(ph[1]); return -3; }
    const int dense = (bits & 6) != 0, energy = (bits & 4) != 0;
    const int Pa = sp[0].P, Pb = sp[1].P;
    const int n_s[2] = {na, nb};
    const int64_t* off[2] = {off_a, off_b};
    const int* holes[2] = {holes_a, holes_b};
    const int* parts[2] = {parts_a, parts_b};
    WS w[2];
    for (int s = 0; s < 2; s++) {
        const int P = sp[s].P;
        w[s].theta = (cd*)malloc(sizeof(cd) * ((size_t)N * n_s[s] + 1));
        w[s].g = (cd*)malloc(sizeof(cd) * (P + 1));
        w[s].B = (cd*)malloc(sizeof(cd) * ((size_t)(ng + 1) * P + 1));
        w[s].X0 = (cd*)malloc(sizeof(cd) * (ng + 1));
        w[s].FK = (cd*)malloc(sizeof(cd) * (P + 1));
        w[s].F = (cd*)malloc(sizeof(cd) * (P + 1));
    }
    cd* Vab = (cd*)malloc(sizeof(cd) * ((size_t)Pa * Pb + 1));
    cd* Vss[2] = {(cd*)malloc(sizeof(cd) * ((size_t)Pa * Pa + 1)), (cd*)malloc(sizeof(cd) * ((size_t)Pb * Pb + 1))};
    const int PT = Pa + Pb;
    for (int iw = 0; iw < nw; iw++) {
        const cd* psi[2] = {phi_a + (size_t)iw * N * na, phi_b + (size_t)iw * N * nb};
        int bad = reference(&sp[0], N, psi[0], &w[0]) | reference(&sp[1], N, psi[1], &w[1]);
        if (bad) {
            if (bits & 1) ovlp[iw] = NAN;
            if (bits & 2) for (int g = 0; g < ng; g++) fb[(size_t)iw * ng + g] = NAN;
            if (energy) for (int t = 0; t < 3; t++) E[iw * 3 + t] = NAN;
            continue;
        }
        if (dense) { half_rotate(&sp[0], N, ng, h1, L, &w[0]); half_rotate(&sp[1], N, ng, h1, L, &w[1]); }
        if (energy) {
            for (int s = 0; s < 2; s++)
                for (int x = 0; x < sp[s].P; x++) {
                    cd t = -w[s].FK[x];
                    for (int g = 0; g < ng; g++) t += (w[0].X0[g] + w[1].X0[g]) * w[s].B[(size_t)g * sp[s].P + x];
                    w[s].F[x] = t;
                }
            vtensor(ng, Pa, Pb, w[0].B, w[1].B, Vab);
            vtensor(ng, Pa, Pa, w[0].B, w[0].B, Vss[0]);
            vtensor(ng, Pb, Pb, w[1].B, w[1].B, Vss[1]);
        }
        /* determinant loop: W2-W4 and the second-order part of W9 */
        cd W = 0.0, E2nd = 0.0;
        cd* C = (cd*)calloc(PT + 1, sizeof(cd));
#pragma omp parallel
        {
            cd lW = 0.0, lE = 0.0;
            cd* lC = (cd*)calloc(PT + 1, sizeof(cd));
#pragma omp for schedule(dynamic, 256)
            for (int64_t d = 0; d < nd; d++) {
                int k[2], x[2][KMAX * KMAX];
                cd A[2][KMAX * KMAX], R[2];
                for (int s = 0; s < 2; s++) {
                    k[s] = (int)(off[s][d + 1] - off[s][d]);
                    R[s] = spin_det(&sp[s], k[s], holes[s] + off[s][d], parts[s] + off[s][d], w[s].g, x[s], A[s]);
                }
                const double ct = ci[d] * ph[0][d] * ph[1][d];
                lW += ct * R[0] * R[1];
                if (dense)
                    for (int s = 0; s < 2; s++) {
                        const cd f = ct * R[1 - s];
                        cd* c = lC + (s ? Pa : 0);
                        for (int a = 0; a < k[s]; a++)
                            for (int b = 0; b < k[s]; b++) c[x[s][a * k[s] + b]] += f * A[s][b * k[s] + a];
                    }
                if (energy) {
                    cd e = 0.0;
                    for (int a = 0; a < k[0]; a++)
                        for (int b = 0; b < k[0]; b++) {
                            const cd* vrow = Vab + (size_t)x[0][a * k[0] + b] * Pb;
                            cd z = 0.0;
                            for (int a2 = 0; a2 < k[1]; a2++)
                                for (int b2 = 0; b2 < k[1]; b2++) z += A[1][b2 * k[1] + a2] * vrow[x[1][a2 * k[1] + b2]];
                            e += A[0][b * k[0] + a] * z;
                        }
                    for (int s = 0; s < 2; s++) {
                        const int ks = k[s], P = sp[s].P;
                        if (ks < 2) continue;
                        cd ess = 0.0;
                        for (int a = 0; a < ks; a++)
                            for (int c = a + 1; c < ks; c++)
                                for (int b = 0; b < ks; b++)
                                    for (int dd = b + 1; dd < ks; dd++) {
                                        cd T = 1.0;
                                        if (ks > 2) {
                                            if (R[s] == 0.0) continue;
                                            T = (A[s][b * ks + a] * A[s][dd * ks + c] - A[s][b * ks + c] * A[s][dd * ks + a]) / R[s];
                                        }
                                        const cd v = Vss[s][(size_t)x[s][a * ks + b] * P + x[s][c * ks + dd]] -
                                                     Vss[s][(size_t)x[s][a * ks + dd] * P + x[s][c * ks + b]];
                                        ess += T * v;
                                    }
                        e += R[1 - s] * ess;
                    }
                    lE += ct * e;
                }
            }
#pragma omp critical
            {
                W += lW; E2nd += lE;
                for (int t = 0; t < PT; t++) C[t] += lC[t];
            }
            free(lC);
        }
        if (bits & 1) ovlp[iw] = w[0].det0 * w[1].det0 * W;
        if (W == 0.0) {
            if (bits & 2) for (int g = 0; g < ng; g++) fb[(size_t)iw * ng + g] = NAN;
            if (energy) for (int t = 0; t < 3; t++) E[iw * 3 + t] = NAN;
            free(C);
            continue;
        }
        if (bits & 2)
            for (int g = 0; g < ng; g++) {
                cd t = 0.0;
                for (int s = 0; s < 2; s++) {
                    const cd* c = C + (s ? Pa : 0);
                    const cd* Bg = w[s].B + (size_t)g * sp[s].P;
                    for (int x = 0; x < sp[s].P; x++) t += c[x] * Bg[x];
                }
                fb[(size_t)iw * ng + g] = w[0].X0[g] + w[1].X0[g] + t / W;
            }
        if (energy) {
            cd ch = 0.0, cf = 0.0, xx = 0.0;
            for (int s = 0; s < 2; s++) {
                const cd* c = C + (s ? Pa : 0);
                const cd* H = w[s].B + (size_t)ng * sp[s].P;
                for (int x = 0; x < sp[s].P; x++) { ch += c[x] * H[x]; cf += c[x] * w[s].F[x]; }
            }
            for (int g = 0; g < ng; g++) { cd xt = w[0].X0[g] + w[1].X0[g]; xx += xt * xt; }
            const cd E1 = w[0].e1_0 + w[1].e1_0 + ch / W;
            const cd E2 = 0.5 * (xx - w[0].ex0 - w[1].ex0) + (cf + E2nd) / W;
            E[iw * 3 + 0] = e0 + E1 + E2; E[iw * 3 + 1] = E1; E[iw * 3 + 2] = E2;
        }
        free(C);
    }
    for (int s = 0; s < 2; s++) { free(w[s].theta); free(w[s].g); free(w[s].B); free(w[s].X0); free(w[s].FK); free(w[s].F); free(Vss[s]); }
    free(Vab); free(sp); free(ph[0]); free(ph[1]);
    return 0;
}

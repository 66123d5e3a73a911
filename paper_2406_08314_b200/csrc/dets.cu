// S2 minors + S3 cofactors + S4 CI reduction + S8 per-determinant energy; the paper's
// get_dets / build_det_matrix / build_cofactor_matrix / reduce_CI / fill_os / get_ss,
// fused: nothing of size (N_w, N_d) or (N_w, N_d, N_gamma) is ever materialised (PAPER.md:L313 chunking is
// unnecessary).  Wick steps W2-W4 and the second-order part of W9.
//
// Thread mapping: a warp = 4 determinants x 8 walkers (MSD_WT); the walker index is the fastest dimension of
// g, C and V, so every gather / atomic of a determinant touches one 128-byte line per 8-walker group.
//   M[a][b] = g[h_a, p_b]                       k x k minor of the reference Green's function
//   R = det M,  A = adj M (A[b][a] = cofactor of M[a][b]),  T[b,d;a,c] = signed complementary (k-2) minor
//   W      += c~ R^a R^b
//   C^s[x] += c~ R^sbar A^s[b][a]               x = (p_b, h_a)
//   E2nd   += c~ [ sum A^a[b][a] A^b[b'][a'] Vab[x][x'] + sum_s R^sbar sum_{a<c,b<d} T^s (Vss[x_ab][x_cd] - Vss[x_ad][x_cb]) ]
// Levels <= 4 use division-free closed forms in registers (exact for singular minors: pin P7);
// higher levels use in-place Gauss-Jordan with partial pivoting in shared memory (one matrix per thread).
#include "msd_internal.cuh"

struct DetsParams {
    const unsigned char* tab;
    const double* coef;
    const cplx* g[2];      // [nt][P][WT]
    cplx* C[2];            // [nt][P][WT]
    const cplx* Vab;       // [nt][Pa][Pb][WT]
    const cplx* Vss[2];    // [nt][P][P][WT]
    cplx* Wacc;            // [nt*WT]
    cplx* E2nd;            // [nt*WT]
    int no[2], P[2];
};

// ------------------------------------------------------------------------------------------------
// closed forms, K <= 4
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ cplx minor2(cplx a, cplx b, cplx c, cplx d) {   // a d - b c
    cplx r = cmul(a, d);
    return cfms(b, c, r);
}

template <int K> struct Closed;

template <> struct Closed<0> {
    __device__ static __forceinline__ cplx det_adj(const cplx (*)[1], cplx (*)[1]) { return cmake(1.0, 0.0); }
};
template <> struct Closed<1> {
    __device__ static __forceinline__ cplx det_adj(const cplx (*M)[1], cplx (*A)[1]) {
        A[0][0] = cmake(1.0, 0.0);
        return M[0][0];
    }
};
template <> struct Closed<2> {
    __device__ static __forceinline__ cplx det_adj(const cplx (*M)[2], cplx (*A)[2]) {
        A[0][0] = M[1][1]; A[0][1] = cneg(M[0][1]);
        A[1][0] = cneg(M[1][0]); A[1][1] = M[0][0];
        return minor2(M[0][0], M[0][1], M[1][0], M[1][1]);
    }
};
template <> struct Closed<3> {
    __device__ static __forceinline__ cplx det_adj(const cplx (*M)[3], cplx (*A)[3]) {
#pragma unroll
        for (int a = 0; a < 3; a++) {
            const int r1 = (a == 0) ? 1 : 0, r2 = (a == 2) ? 1 : 2;
#pragma unroll
            for (int b = 0; b < 3; b++) {
                const int c1 = (b == 0) ? 1 : 0, c2 = (b == 2) ? 1 : 2;
                cplx m = minor2(M[r1][c1], M[r1][c2], M[r2][c1], M[r2][c2]);
                A[b][a] = ((a + b) & 1) ? cneg(m) : m;
            }
        }
        cplx R = cmul(M[0][0], A[0][0]);
        R = cfma(M[0][1], A[1][0], R);
        R = cfma(M[0][2], A[2][0], R);
        return R;
    }
};
// pair index of columns (i<j) of a 4-wide matrix: 01->0 02->1 03->2 12->3 13->4 23->5
__device__ __forceinline__ constexpr int pidx4(int i, int j) { return i == 0 ? j - 1 : (i == 1 ? j + 1 : 5); }
template <> struct Closed<4> {
    __device__ static __forceinline__ cplx det_adj(const cplx (*M)[4], cplx (*A)[4]) {
        cplx s[6], c[6];   // 2x2 minors of rows (0,1) and of rows (2,3)
#pragma unroll
        for (int i = 0; i < 4; i++)
#pragma unroll
            for (int j = i + 1; j < 4; j++) {
                s[pidx4(i, j)] = minor2(M[0][i], M[0][j], M[1][i], M[1][j]);
                c[pidx4(i, j)] = minor2(M[2][i], M[2][j], M[3][i], M[3][j]);
            }
        cplx R = cmul(s[0], c[5]);
        R = cfms(s[1], c[4], R);
        R = cfma(s[2], c[3], R);
        R = cfma(s[3], c[2], R);
        R = cfms(s[4], c[1], R);
        R = cfma(s[5], c[0], R);
#pragma unroll
        for (int a = 0; a < 4; a++) {
            // 3x3 minor with row a deleted = the surviving row t of a's pair times 2x2 minors of the other pair.
            // Row t is the first row (a<2: rows t,2,3) or the last row (a>=2: rows 0,1,t) of the 3x3 minor;
            // both expand with signs + - +.
            const int t = (a < 2) ? 1 - a : 5 - a;
#pragma unroll
            for (int b = 0; b < 4; b++) {
                const int j1 = (b == 0) ? 1 : 0, j2 = (b <= 1) ? 2 : 1, j3 = (b == 3) ? 2 : 3;
                cplx m;
                if (a < 2) {
                    m = cmul(M[t][j1], c[pidx4(j2, j3)]);
                    m = cfms(M[t][j2], c[pidx4(j1, j3)], m);
                    m = cfma(M[t][j3], c[pidx4(j1, j2)], m);
                } else {
                    m = cmul(M[t][j1], s[pidx4(j2, j3)]);
                    m = cfms(M[t][j2], s[pidx4(j1, j3)], m);
                    m = cfma(M[t][j3], s[pidx4(j1, j2)], m);
                }
                A[b][a] = ((a + b) & 1) ? cneg(m) : m;   // cofactor sign (-1)^(a+b)
            }
        }
        return R;
    }
};

// second-order cofactor T[b,d;a,c], a<c, b<d: (-1)^(a+b+c+d) det(M without rows a,c and columns b,d)
template <int K>
__device__ __forceinline__ cplx second_cofactor(const cplx (*M)[K > 0 ? K : 1], int a, int c, int b, int d)
{
    if (K == 2) return cmake(1.0, 0.0);
    cplx m;
    if (K == 3) {
        const int r = 3 - a - c, q = 3 - b - d;
        m = M[r][q];
    } else {   // K == 4: the two surviving rows / columns, ascending (a<c, b<d)
        const int r1 = (a > 0) ? 0 : ((c > 1) ? 1 : 2), r2 = (c < 3) ? 3 : ((a < 2) ? 2 : 1);
        const int c1 = (b > 0) ? 0 : ((d > 1) ? 1 : 2), c2 = (d < 3) ? 3 : ((b < 2) ? 2 : 1);
        m = minor2(M[r1][c1], M[r1][c2], M[r2][c1], M[r2][c2]);
    }
    return ((a + b + c + d) & 1) ? cneg(m) : m;
}

// one spin of one (determinant, walker): gather, det, adjugate, same-spin second-order sum
template <int K, int MODE>
struct SpinEval {
    cplx A[K > 0 ? K : 1][K > 0 ? K : 1];
    int x[K > 0 ? K : 1][K > 0 ? K : 1];     // pair index x[a][b] = p_b * n_o + h_a
    cplx R;
    cplx Ess;
    __device__ __forceinline__ void run(const unsigned char* hp, const cplx* __restrict__ g, int no,
                                        const cplx* __restrict__ Vss, int P)
    {
        Ess = cmake(0.0, 0.0);
        if (K == 0) { R = cmake(1.0, 0.0); return; }
        cplx M[K > 0 ? K : 1][K > 0 ? K : 1];
#pragma unroll
        for (int a = 0; a < K; a++)
#pragma unroll
            for (int b = 0; b < K; b++) {
                x[a][b] = (int)hp[K + b] * no + (int)hp[a];
                M[a][b] = __ldg(&g[(int64_t)x[a][b] * MSD_WT]);
            }
        R = Closed<K>::det_adj(M, A);
        if (MODE == 2 && K >= 2) {
#pragma unroll
            for (int a = 0; a < K; a++)
#pragma unroll
                for (int c = a + 1; c < K; c++)
#pragma unroll
                    for (int b = 0; b < K; b++)
#pragma unroll
                        for (int d = b + 1; d < K; d++) {
                            cplx t = second_cofactor<K>(M, a, c, b, d);
                            cplx v1 = __ldg(&Vss[((int64_t)x[a][b] * P + x[c][d]) * MSD_WT]);
                            cplx v2 = __ldg(&Vss[((int64_t)x[a][d] * P + x[c][b]) * MSD_WT]);
                            Ess = cfma(t, csub(v1, v2), Ess);
                        }
        }
    }
};

template <int KA, int KB, int MODE>
__device__ __forceinline__ void run_bucket(const DetsParams& p, const WorkItem& it, int tile, int slot, int nslots,
                                           int j, cplx& Wl, cplx& El)
{
    constexpr int NB = 2 * KA + 2 * KB;
    constexpr int NWORD = (NB + 3) / 4 > 0 ? (NB + 3) / 4 : 1;
    const cplx* gA = p.g[0] + (int64_t)tile * p.P[0] * MSD_WT + j;
    const cplx* gB = p.g[1] + (int64_t)tile * p.P[1] * MSD_WT + j;
    cplx* CA = p.C[0] + (int64_t)tile * p.P[0] * MSD_WT + j;
    cplx* CB = p.C[1] + (int64_t)tile * p.P[1] * MSD_WT + j;
    const cplx* VA = (MODE == 2) ? p.Vss[0] + (int64_t)tile * p.P[0] * p.P[0] * MSD_WT + j : nullptr;
    const cplx* VB = (MODE == 2) ? p.Vss[1] + (int64_t)tile * p.P[1] * p.P[1] * MSD_WT + j : nullptr;
    const cplx* VAB = (MODE == 2) ? p.Vab + (int64_t)tile * p.P[0] * p.P[1] * MSD_WT + j : nullptr;
    for (int i = slot; i < it.det_count; i += nslots) {
        union { uint32_t w[NWORD]; unsigned char b[NWORD * 4]; } row;
        const uint32_t* rp = reinterpret_cast<const uint32_t*>(p.tab + it.tab_off + (int64_t)i * it.rs);
#pragma unroll
        for (int t = 0; t < NWORD; t++) row.w[t] = (NB > 0) ? __ldg(rp + t) : 0u;
        const double cf = __ldg(&p.coef[it.det_begin + i]);
        SpinEval<KA, MODE> ea;
        SpinEval<KB, MODE> eb;
        ea.run(row.b, gA, p.no[0], VA, p.P[0]);
        eb.run(row.b + 2 * KA, gB, p.no[1], VB, p.P[1]);
        const cplx cRa = cscale(cf, ea.R), cRb = cscale(cf, eb.R);
        Wl = cfma(cRa, eb.R, Wl);
        if (MODE >= 1) {
#pragma unroll
            for (int a = 0; a < KA; a++)
#pragma unroll
                for (int b = 0; b < KA; b++) red_add(&CA[(int64_t)ea.x[a][b] * MSD_WT], cmul(cRb, ea.A[b][a]));
#pragma unroll
            for (int a = 0; a < KB; a++)
#pragma unroll
                for (int b = 0; b < KB; b++) red_add(&CB[(int64_t)eb.x[a][b] * MSD_WT], cmul(cRa, eb.A[b][a]));
        }
        if (MODE == 2) {
            cplx e = cmake(0.0, 0.0);
            if (KA > 0 && KB > 0) {
#pragma unroll
                for (int a = 0; a < KA; a++)
#pragma unroll
                    for (int b = 0; b < KA; b++) {
                        const cplx* vrow = VAB + (int64_t)ea.x[a][b] * p.P[1] * MSD_WT;
                        cplx z = cmake(0.0, 0.0);
#pragma unroll
                        for (int a2 = 0; a2 < KB; a2++)
#pragma unroll
                            for (int b2 = 0; b2 < KB; b2++)
                                z = cfma(eb.A[b2][a2], __ldg(&vrow[(int64_t)eb.x[a2][b2] * MSD_WT]), z);
                        e = cfma(ea.A[b][a], z, e);
                    }
            }
            e = cfma(eb.R, ea.Ess, e);
            e = cfma(ea.R, eb.Ess, e);
            El.x = fma(cf, e.x, El.x);
            El.y = fma(cf, e.y, El.y);
        }
    }
}

// reduce per-lane partial sums over the CTA's determinant slots and add to the walker accumulators
__device__ __forceinline__ void flush_walker_sums(const DetsParams& p, int tile, cplx Wl, cplx El, int mode)
{
    __shared__ double acc[MSD_WT][4];
    double v[4] = {Wl.x, Wl.y, El.x, El.y};
#pragma unroll
    for (int t = 0; t < 4; t++) {      // the 4 determinant slots of a warp share each walker lane j
        v[t] += __shfl_xor_sync(0xffffffffu, v[t], 8);
        v[t] += __shfl_xor_sync(0xffffffffu, v[t], 16);
    }
    if (threadIdx.x < MSD_WT * 4) acc[threadIdx.x >> 2][threadIdx.x & 3] = 0.0;
    __syncthreads();
    const int lane = threadIdx.x & 31;
    if (lane < MSD_WT) {
#pragma unroll
        for (int t = 0; t < 4; t++) atomicAdd(&acc[lane][t], v[t]);
    }
    __syncthreads();
    if (threadIdx.x < MSD_WT) {
        const int jj = threadIdx.x;
        atomicAdd(&p.Wacc[tile * MSD_WT + jj].x, acc[jj][0]);
        atomicAdd(&p.Wacc[tile * MSD_WT + jj].y, acc[jj][1]);
        if (mode == 2) {
            atomicAdd(&p.E2nd[tile * MSD_WT + jj].x, acc[jj][2]);
            atomicAdd(&p.E2nd[tile * MSD_WT + jj].y, acc[jj][3]);
        }
    }
}

#define CF_CASE(KA_, KB_)                                                                              \
    case KA_ * 5 + KB_:                                                                                \
        if constexpr ((KA_ > KB_ ? KA_ : KB_) > KLO && (KA_ > KB_ ? KA_ : KB_) <= KHI)                  \
            run_bucket<KA_, KB_, MODE>(p, it, tile, slot, nslots, j, Wl, El);                          \
        break;

// register class (KLO, KHI]: buckets whose larger level lies in that range (KLO = -1 admits (0,0))
template <int MODE, int KLO, int KHI>
__global__ void __launch_bounds__(128) k_dets_cf(DetsParams p, const WorkItem* __restrict__ items)
{
    const WorkItem it = items[blockIdx.x];
    const int tile = blockIdx.y;
    const int j = threadIdx.x & (MSD_WT - 1);
    const int slot = threadIdx.x / MSD_WT, nslots = blockDim.x / MSD_WT;
    cplx Wl = cmake(0.0, 0.0), El = cmake(0.0, 0.0);
    switch (it.ka * 5 + it.kb) {
        CF_CASE(0, 0) CF_CASE(0, 1) CF_CASE(0, 2) CF_CASE(0, 3) CF_CASE(0, 4)
        CF_CASE(1, 0) CF_CASE(1, 1) CF_CASE(1, 2) CF_CASE(1, 3) CF_CASE(1, 4)
        CF_CASE(2, 0) CF_CASE(2, 1) CF_CASE(2, 2) CF_CASE(2, 3) CF_CASE(2, 4)
        CF_CASE(3, 0) CF_CASE(3, 1) CF_CASE(3, 2) CF_CASE(3, 3) CF_CASE(3, 4)
        CF_CASE(4, 0) CF_CASE(4, 1) CF_CASE(4, 2) CF_CASE(4, 3) CF_CASE(4, 4)
        default: break;
    }
    flush_walker_sums(p, tile, Wl, El, MODE);
}

// ------------------------------------------------------------------------------------------------
// generic levels (k >= 5 in at least one spin): one matrix per thread in shared memory, element e of
// thread t at sm[e * T + t]
// ------------------------------------------------------------------------------------------------
struct SmMat {
    cplx* base; int T;
    __device__ __forceinline__ cplx& at(int e) { return base[(int64_t)e * T]; }
};

// in-place Gauss-Jordan inverse with partial pivoting; returns det (0 if an exactly zero pivot appears,
// in which case the matrix content is zeroed: adj and second cofactors are taken as 0 -- reading A11)
__device__ cplx gauss_jordan(SmMat m, int k)
{
    int ipiv[MSD_MAX_LEVEL];
    cplx det = cmake(1.0, 0.0);
    bool sing = false;
    for (int j = 0; j < k; j++) {
        int p = j; double best = cabs2(m.at(j * k + j));
        for (int i = j + 1; i < k; i++) { double v = cabs2(m.at(i * k + j)); if (v > best) { best = v; p = i; } }
        ipiv[j] = p;
        if (!(best > 0.0)) { sing = true; break; }
        if (p != j) {
            for (int c = 0; c < k; c++) { cplx t = m.at(j * k + c); m.at(j * k + c) = m.at(p * k + c); m.at(p * k + c) = t; }
            det = cneg(det);
        }
        cplx pv = m.at(j * k + j);
        det = cmul(det, pv);
        cplx r = cinv(pv);
        m.at(j * k + j) = cmake(1.0, 0.0);
        for (int c = 0; c < k; c++) m.at(j * k + c) = cmul(m.at(j * k + c), r);
        for (int i = 0; i < k; i++) {
            if (i == j) continue;
            cplx f = m.at(i * k + j);
            m.at(i * k + j) = cmake(0.0, 0.0);
            for (int c = 0; c < k; c++) m.at(i * k + c) = cfms(f, m.at(j * k + c), m.at(i * k + c));
        }
    }
    if (sing) {
        for (int e = 0; e < k * k; e++) m.at(e) = cmake(0.0, 0.0);
        return cmake(0.0, 0.0);
    }
    for (int j = k - 1; j >= 0; j--) {
        int p = ipiv[j];
        if (p != j)
            for (int i = 0; i < k; i++) { cplx t = m.at(i * k + j); m.at(i * k + j) = m.at(i * k + p); m.at(i * k + p) = t; }
    }
    return det;
}

template <int K>
__device__ __forceinline__ cplx closed_to_smem(SmMat m, cplx* Ess, const int* x, const cplx* __restrict__ Vss, int P,
                                               int mode)
{
    cplx M[K][K], A[K][K];
#pragma unroll
    for (int a = 0; a < K; a++)
#pragma unroll
        for (int b = 0; b < K; b++) M[a][b] = m.at(a * K + b);
    cplx R = Closed<K>::det_adj(M, A);
#pragma unroll
    for (int a = 0; a < K; a++)
#pragma unroll
        for (int b = 0; b < K; b++) m.at(b * K + a) = A[b][a];
    cplx e = cmake(0.0, 0.0);
    if (mode == 2 && K >= 2) {
#pragma unroll
        for (int a = 0; a < K; a++)
#pragma unroll
            for (int c = a + 1; c < K; c++)
#pragma unroll
                for (int b = 0; b < K; b++)
#pragma unroll
                    for (int d = b + 1; d < K; d++) {
                        cplx t = second_cofactor<K>(M, a, c, b, d);
                        cplx v1 = __ldg(&Vss[((int64_t)x[a * K + b] * P + x[c * K + d]) * MSD_WT]);
                        cplx v2 = __ldg(&Vss[((int64_t)x[a * K + d] * P + x[c * K + b]) * MSD_WT]);
                        e = cfma(t, csub(v1, v2), e);
                    }
    }
    *Ess = e;
    return R;
}

// one spin, runtime level k; on exit m holds A (A[b][a] at element b*k+a), returns R, *Ess
__device__ cplx spin_generic(SmMat m, int k, const unsigned char* hp, const cplx* __restrict__ g, int no, int* x,
                             const cplx* __restrict__ Vss, int P, int mode, cplx* Ess)
{
    *Ess = cmake(0.0, 0.0);
    if (k == 0) return cmake(1.0, 0.0);
    for (int a = 0; a < k; a++)
        for (int b = 0; b < k; b++) {
            int xx = (int)hp[k + b] * no + (int)hp[a];
            x[a * k + b] = xx;
            m.at(a * k + b) = __ldg(&g[(int64_t)xx * MSD_WT]);
        }
    switch (k) {
        case 1: return closed_to_smem<1>(m, Ess, x, Vss, P, mode);
        case 2: return closed_to_smem<2>(m, Ess, x, Vss, P, mode);
        case 3: return closed_to_smem<3>(m, Ess, x, Vss, P, mode);
        case 4: return closed_to_smem<4>(m, Ess, x, Vss, P, mode);
        default: break;
    }
    cplx R = gauss_jordan(m, k);          // m = M^-1 (or zeros)
    for (int e = 0; e < k * k; e++) m.at(e) = cmul(R, m.at(e));   // A = R M^-1
    if (mode == 2 && (R.x != 0.0 || R.y != 0.0)) {
        // T[b,d;a,c] = R (Minv[b][a] Minv[d][c] - Minv[b][c] Minv[d][a]) = (A[b][a] A[d][c] - A[b][c] A[d][a]) / R
        cplx e = cmake(0.0, 0.0);
        for (int a = 0; a < k; a++)
            for (int c = a + 1; c < k; c++)
                for (int b = 0; b < k; b++)
                    for (int d = b + 1; d < k; d++) {
                        cplx t = cmul(m.at(b * k + a), m.at(d * k + c));
                        t = cfms(m.at(b * k + c), m.at(d * k + a), t);
                        cplx v1 = __ldg(&Vss[((int64_t)x[a * k + b] * P + x[c * k + d]) * MSD_WT]);
                        cplx v2 = __ldg(&Vss[((int64_t)x[a * k + d] * P + x[c * k + b]) * MSD_WT]);
                        e = cfma(t, csub(v1, v2), e);
                    }
        *Ess = cmul(e, cinv(R));
    }
    return R;
}

template <int MODE>
__global__ void k_dets_gen(DetsParams p, const WorkItem* __restrict__ items, int smem_elems_per_thread)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const WorkItem it = items[blockIdx.x];
    const int tile = blockIdx.y;
    const int j = threadIdx.x & (MSD_WT - 1);
    const int slot = threadIdx.x / MSD_WT, nslots = blockDim.x / MSD_WT;
    const int T = blockDim.x;
    cplx* sm = reinterpret_cast<cplx*>(smem_raw) + threadIdx.x;
    (void)smem_elems_per_thread;
    const int ka = it.ka, kb = it.kb;
    SmMat mA{sm, T}, mB{sm + (int64_t)ka * ka * T, T};
    const cplx* gA = p.g[0] + (int64_t)tile * p.P[0] * MSD_WT + j;
    const cplx* gB = p.g[1] + (int64_t)tile * p.P[1] * MSD_WT + j;
    cplx* CA = p.C[0] + (int64_t)tile * p.P[0] * MSD_WT + j;
    cplx* CB = p.C[1] + (int64_t)tile * p.P[1] * MSD_WT + j;
    const cplx* VA = (MODE == 2) ? p.Vss[0] + (int64_t)tile * p.P[0] * p.P[0] * MSD_WT + j : nullptr;
    const cplx* VB = (MODE == 2) ? p.Vss[1] + (int64_t)tile * p.P[1] * p.P[1] * MSD_WT + j : nullptr;
    const cplx* VAB = (MODE == 2) ? p.Vab + (int64_t)tile * p.P[0] * p.P[1] * MSD_WT + j : nullptr;
    cplx Wl = cmake(0.0, 0.0), El = cmake(0.0, 0.0);
    int xa[MSD_MAX_LEVEL * MSD_MAX_LEVEL], xb[MSD_MAX_LEVEL * MSD_MAX_LEVEL];
    for (int i = slot; i < it.det_count; i += nslots) {
        const unsigned char* row = p.tab + it.tab_off + (int64_t)i * it.rs;
        unsigned char hp[4 * MSD_MAX_LEVEL];
        for (int t = 0; t < 2 * ka + 2 * kb; t++) hp[t] = __ldg(row + t);
        const double cf = __ldg(&p.coef[it.det_begin + i]);
        cplx EssA, EssB;
        cplx Ra = spin_generic(mA, ka, hp, gA, p.no[0], xa, VA, p.P[0], MODE, &EssA);
        cplx Rb = spin_generic(mB, kb, hp + 2 * ka, gB, p.no[1], xb, VB, p.P[1], MODE, &EssB);
        const cplx cRa = cscale(cf, Ra), cRb = cscale(cf, Rb);
        Wl = cfma(cRa, Rb, Wl);
        if (MODE >= 1) {
            for (int a = 0; a < ka; a++)
                for (int b = 0; b < ka; b++) red_add(&CA[(int64_t)xa[a * ka + b] * MSD_WT], cmul(cRb, mA.at(b * ka + a)));
            for (int a = 0; a < kb; a++)
                for (int b = 0; b < kb; b++) red_add(&CB[(int64_t)xb[a * kb + b] * MSD_WT], cmul(cRa, mB.at(b * kb + a)));
        }
        if (MODE == 2) {
            cplx e = cmake(0.0, 0.0);
            for (int a = 0; a < ka; a++)
                for (int b = 0; b < ka; b++) {
                    const cplx* vrow = VAB + (int64_t)xa[a * ka + b] * p.P[1] * MSD_WT;
                    cplx z = cmake(0.0, 0.0);
                    for (int a2 = 0; a2 < kb; a2++)
                        for (int b2 = 0; b2 < kb; b2++)
                            z = cfma(mB.at(b2 * kb + a2), __ldg(&vrow[(int64_t)xb[a2 * kb + b2] * MSD_WT]), z);
                    e = cfma(mA.at(b * ka + a), z, e);
                }
            e = cfma(Rb, EssA, e);
            e = cfma(Ra, EssB, e);
            El.x = fma(cf, e.x, El.x);
            El.y = fma(cf, e.y, El.y);
        }
    }
    flush_walker_sums(p, tile, Wl, El, MODE);
}

// ------------------------------------------------------------------------------------------------
template <int MODE>
static cudaError_t launch_mode(msd_ctx* c, const DetsParams& p, int ntiles, cudaStream_t st)
{
    // three register classes of the closed-form kernel, split on the host by the items' larger level
    const WorkItem* d = c->d_items_cf;
    size_t n = c->items_cf.size();
    size_t i0 = 0;
    // items_cf is sorted by class (ascending larger level), see build_work_items()
    auto cls = [&](const WorkItem& w) { int m = w.ka > w.kb ? w.ka : w.kb; return m <= 2 ? 0 : (m == 3 ? 1 : 2); };
    while (i0 < n) {
        size_t i1 = i0; int cl = cls(c->items_cf[i0]);
        while (i1 < n && cls(c->items_cf[i1]) == cl) i1++;
        dim3 grid((unsigned)(i1 - i0), ntiles);
        if (cl == 0) k_dets_cf<MODE, -1, 2><<<grid, 128, 0, st>>>(p, d + i0);
        else if (cl == 1) k_dets_cf<MODE, 2, 3><<<grid, 128, 0, st>>>(p, d + i0);
        else k_dets_cf<MODE, 3, 4><<<grid, 128, 0, st>>>(p, d + i0);
        c->launches++;
        i0 = i1;
    }
    if (!c->items_gen.empty()) {
        size_t smem = (size_t)c->gen_smem_per_thread * c->gen_threads;
        cudaError_t e = cudaFuncSetAttribute(k_dets_gen<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        dim3 grid((unsigned)c->items_gen.size(), ntiles);
        k_dets_gen<MODE><<<grid, c->gen_threads, smem, st>>>(p, c->d_items_gen, c->gen_smem_per_thread / 16);
        c->launches++;
    }
    return cudaGetLastError();
}

cudaError_t launch_dets(msd_ctx* c, int mode, int64_t nw, Workspace& ws, cudaStream_t st)
{
    DetsParams p;
    p.tab = c->d_tab; p.coef = c->d_coef;
    for (int s = 0; s < 2; s++) {
        p.g[s] = ws.g[s]; p.C[s] = ws.C[s]; p.Vss[s] = ws.Vss[s];
        p.no[s] = c->sp[s].n_o; p.P[s] = c->sp[s].P;
    }
    p.Vab = ws.Vab; p.Wacc = ws.Wacc; p.E2nd = ws.E2nd;
    int ntiles = (int)((nw + MSD_WT - 1) / MSD_WT);
    if (mode == 0) return launch_mode<0>(c, p, ntiles, st);
    if (mode == 1) return launch_mode<1>(c, p, ntiles, st);
    return launch_mode<2>(c, p, ntiles, st);
}

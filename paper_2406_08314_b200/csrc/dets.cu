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
//   C^s[x] += c~ R^sbar A^s[b][a]               x = (p_b, h_a)      (overlap / force-bias modes: RED.ADD.F64 scatter)
//   energy mode needs C only inside sum_x C[x] Hrot[x] and sum_x C[x] F[x], so those two scalars are accumulated
//   per determinant from gathers of Hrot / F (two 128-byte lines per entry) and C is never formed: no atomics.
//   E2nd   += c~ [ sum A^a[b][a] A^b[b'][a'] Vab[x][x'] + sum_s R^sbar sum_{a<c,b<d} T^s Vbar^s[x_ab][x_cd] ]
//   Vbar^s[x_ab][x_cd] = V^ss[x_ab][x_cd] - V^ss[x_ad][x_cb]  (k_vbar, in place on the h_a<h_c, p_b<p_d entries of Vss)
// Levels <= 4 use division-free closed forms in registers (exact for singular minors: pin P7);
// higher levels use in-place Gauss-Jordan with partial pivoting in shared memory (one matrix per thread).
#include "msd_internal.cuh"
// MODE: 0 overlap (W only), 1 force bias (W, C scatter), 2 energy (W, second-order sums, no C), 3 energy + C scatter
// (the fused force-bias + energy call)
#define M_ENERGY(M) ((M) >= 2)
#define M_SCATTER(M) ((M) == 1 || (M) == 3)
#include <algorithm>

struct DetsParams {
    const unsigned char* tab;
    const double* coef;
    const cplx* g[2];      // [nt][P][WT]
    double* C[2];          // [nt][P][2][WT] planar
    const cplx* Vab;       // [nt][Pa][Pb][WT]
    const cplx* Vss[2];    // [nt][P][P][WT]; entries (h_a<h_c, p_b<p_d) hold the antisymmetrised Vbar (k_vbar)
    const cplx* FH[2];     // [nt][P][2][WT]: Hrot (slot 0) and F (slot 1), walker fastest (k_fh_tile); energy mode only
    cplx* Wacc;            // [nt*WT]
    cplx* E2nd;            // [nt*WT]  second-order two-body sums + sum_x C[x] F[x]
    cplx* E1nd;            // [nt*WT]  sum_x C[x] Hrot[x]
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

// one spin of one (determinant, walker): gather from the shared-memory copy of g, det, adjugate,
// same-spin second-order sum
template <int K, int MODE>
struct SpinEval {
    static constexpr int K1 = K > 0 ? K : 1;
    cplx A[K1][K1];
    int h[K1], pn[K1];                        // h_a and p_b * n_o: pair index x(a,b) = pn[b] + h[a]
    cplx R;
    cplx Ess;
    __device__ __forceinline__ int x(int a, int b) const { return pn[b] + h[a]; }
    __device__ __forceinline__ void run(const unsigned char* hp, const cplx* g /* smem tile + lane walker */, int no,
                                        const cplx* __restrict__ Vss, unsigned P)
    {
        Ess = cmake(0.0, 0.0);
        if (K == 0) { R = cmake(1.0, 0.0); return; }
        cplx M[K1][K1];
#pragma unroll
        for (int a = 0; a < K; a++) { h[a] = (int)hp[a]; pn[a] = (int)hp[K + a] * no; }
#pragma unroll
        for (int a = 0; a < K; a++)
#pragma unroll
            for (int b = 0; b < K; b++) M[a][b] = g[x(a, b) * MSD_WT];
        R = Closed<K>::det_adj(M, A);
        if (M_ENERGY(MODE) && K >= 2) {
#pragma unroll
            for (int a = 0; a < K; a++)
#pragma unroll
                for (int c = a + 1; c < K; c++)
#pragma unroll
                    for (int b = 0; b < K; b++)
#pragma unroll
                        for (int d = b + 1; d < K; d++) {
                            cplx t = second_cofactor<K>(M, a, c, b, d);
                            Ess = cfma(t, __ldg(&Vss[((unsigned)x(a, b) * P + (unsigned)x(c, d)) * MSD_WT]), Ess);
                        }
        }
    }
};

template <int NWORD> struct RowData { uint32_t w[NWORD]; double cf; };

template <int KA, int KB, int MODE, bool FHS>
__device__ __forceinline__ void run_bucket(const DetsParams& p, const WorkItem& it, int tile, int slot, int nslots,
                                           int j, const cplx* gsm, const cplx* gA, const cplx* gB, cplx& Wl, cplx& El, cplx& Hl)
{
    constexpr int NB = 2 * KA + 2 * KB;
    constexpr int NWORD = (NB + 3) / 4 > 0 ? (NB + 3) / 4 : 1;
    double* CA = p.C[0] + (int64_t)tile * p.P[0] * 2 * MSD_WT + j;
    double* CB = p.C[1] + (int64_t)tile * p.P[1] * 2 * MSD_WT + j;
    const cplx* VA = (M_ENERGY(MODE)) ? p.Vss[0] + (int64_t)tile * p.P[0] * p.P[0] * MSD_WT + j : nullptr;
    const cplx* VB = (M_ENERGY(MODE)) ? p.Vss[1] + (int64_t)tile * p.P[1] * p.P[1] * MSD_WT + j : nullptr;
    const cplx* VAB = (M_ENERGY(MODE)) ? p.Vab + (int64_t)tile * p.P[0] * p.P[1] * MSD_WT + j : nullptr;
    // Hrot / F of the tile: the shared-memory copy behind g (FHS) or global memory through L1
    const cplx* FHA = (!M_ENERGY(MODE)) ? nullptr : FHS ? gsm + (p.P[0] + p.P[1]) * MSD_WT + j
                                                  : p.FH[0] + (int64_t)tile * p.P[0] * 2 * MSD_WT + j;
    const cplx* FHB = (!M_ENERGY(MODE)) ? nullptr : FHS ? FHA + p.P[0] * 2 * MSD_WT
                                                  : p.FH[1] + (int64_t)tile * p.P[1] * 2 * MSD_WT + j;
    const unsigned char* tab = p.tab + it.tab_off;
    const double* coef = p.coef + it.det_begin;
    auto load_row = [&](int i, RowData<NWORD>& r) {
        const uint32_t* rp = reinterpret_cast<const uint32_t*>(tab + (int64_t)i * it.rs);
#pragma unroll
        for (int t = 0; t < NWORD; t++) r.w[t] = (NB > 0) ? __ldg(rp + t) : 0u;
        r.cf = __ldg(coef + i);
    };
    int i = slot;
    RowData<NWORD> cur, nxt;
    if (i < it.det_count) load_row(i, cur);
    while (i < it.det_count) {
        const int inext = i + nslots;
        nxt = cur;
        if (inext < it.det_count) load_row(inext, nxt);      // software prefetch of the next table row
        const unsigned char* rb = reinterpret_cast<const unsigned char*>(cur.w);
        const double cf = cur.cf;
        SpinEval<KA, MODE> ea;
        SpinEval<KB, MODE> eb;
        ea.run(rb, gA, p.no[0], VA, (unsigned)p.P[0]);
        eb.run(rb + 2 * KA, gB, p.no[1], VB, (unsigned)p.P[1]);
        const cplx cRa = cscale(cf, ea.R), cRb = cscale(cf, eb.R);
        Wl = cfma(cRa, eb.R, Wl);
        if (M_ENERGY(MODE)) {
            cplx e = cmake(0.0, 0.0);
            if (KA > 0 && KB > 0) {
#pragma unroll
                for (int a = 0; a < KA; a++)
#pragma unroll
                    for (int b = 0; b < KA; b++) {
                        const cplx* vrow = VAB + (unsigned)ea.x(a, b) * (unsigned)p.P[1] * MSD_WT;
                        cplx z = cmake(0.0, 0.0);
#pragma unroll
                        for (int a2 = 0; a2 < KB; a2++)
#pragma unroll
                            for (int b2 = 0; b2 < KB; b2++)
                                z = cfma(eb.A[b2][a2], __ldg(&vrow[eb.x(a2, b2) * MSD_WT]), z);
                        e = cfma(ea.A[b][a], z, e);
                    }
            }
            // sum_x C[x] Hrot[x] and sum_x C[x] F[x] without forming C:  s = sum_ab A[b][a] (Hrot, F)[x_ab]
            cplx shA = cmake(0.0, 0.0), sfA = shA, shB = shA, sfB = shA;
#pragma unroll
            for (int a = 0; a < KA; a++)
#pragma unroll
                for (int b = 0; b < KA; b++) {
                    const cplx* q = FHA + ea.x(a, b) * (2 * MSD_WT);
                    shA = cfma(ea.A[b][a], FHS ? q[0] : __ldg(q), shA);
                    sfA = cfma(ea.A[b][a], FHS ? q[MSD_WT] : __ldg(q + MSD_WT), sfA);
                }
#pragma unroll
            for (int a = 0; a < KB; a++)
#pragma unroll
                for (int b = 0; b < KB; b++) {
                    const cplx* q = FHB + eb.x(a, b) * (2 * MSD_WT);
                    shB = cfma(eb.A[b][a], FHS ? q[0] : __ldg(q), shB);
                    sfB = cfma(eb.A[b][a], FHS ? q[MSD_WT] : __ldg(q + MSD_WT), sfB);
                }
            e = cfma(eb.R, cadd(ea.Ess, sfA), e);
            e = cfma(ea.R, cadd(eb.Ess, sfB), e);
            El.x = fma(cf, e.x, El.x);
            El.y = fma(cf, e.y, El.y);
            cplx hsum = cmul(eb.R, shA);
            hsum = cfma(ea.R, shB, hsum);
            Hl.x = fma(cf, hsum.x, Hl.x);
            Hl.y = fma(cf, hsum.y, Hl.y);
        }
        if (M_SCATTER(MODE)) {
#pragma unroll
            for (int a = 0; a < KA; a++)
#pragma unroll
                for (int b = 0; b < KA; b++) red_add_planar(CA, ea.x(a, b), cmul(cRb, ea.A[b][a]));
#pragma unroll
            for (int a = 0; a < KB; a++)
#pragma unroll
                for (int b = 0; b < KB; b++) red_add_planar(CB, eb.x(a, b), cmul(cRa, eb.A[b][a]));
        }
        cur = nxt;
        i = inext;
    }
}

// reduce per-lane partial sums over the CTA's determinant slots and add to the walker accumulators
__device__ __forceinline__ void flush_walker_sums(const DetsParams& p, int tile, cplx Wl, cplx El, cplx Hl, int mode)
{
    __shared__ double acc[MSD_WT][6];
    double v[6] = {Wl.x, Wl.y, El.x, El.y, Hl.x, Hl.y};
#pragma unroll
    for (int t = 0; t < 6; t++) {      // the 4 determinant slots of a warp share each walker lane j
        v[t] += __shfl_xor_sync(0xffffffffu, v[t], 8);
        v[t] += __shfl_xor_sync(0xffffffffu, v[t], 16);
    }
    for (int t = threadIdx.x; t < MSD_WT * 6; t += blockDim.x) acc[t / 6][t % 6] = 0.0;     // blockDim.x may be 32
    __syncthreads();
    const int lane = threadIdx.x & 31;
    if (lane < MSD_WT) {
#pragma unroll
        for (int t = 0; t < 6; t++) if (t < 2 || mode >= 2) atomicAdd(&acc[lane][t], v[t]);
    }
    __syncthreads();
    if (threadIdx.x < MSD_WT) {
        const int jj = threadIdx.x;
        atomicAdd(&p.Wacc[tile * MSD_WT + jj].x, acc[jj][0]);
        atomicAdd(&p.Wacc[tile * MSD_WT + jj].y, acc[jj][1]);
        if (mode >= 2) {
            atomicAdd(&p.E2nd[tile * MSD_WT + jj].x, acc[jj][2]);
            atomicAdd(&p.E2nd[tile * MSD_WT + jj].y, acc[jj][3]);
            atomicAdd(&p.E1nd[tile * MSD_WT + jj].x, acc[jj][4]);
            atomicAdd(&p.E1nd[tile * MSD_WT + jj].y, acc[jj][5]);
        }
    }
}

// stage the walker tile's active slices g^a, g^b ([P][WT] complex each) in shared memory
__device__ __forceinline__ void stage_g(const DetsParams& p, int tile, cplx* gsm, bool fh)
{
    const int na = p.P[0] * MSD_WT, nb = p.P[1] * MSD_WT;
    const cplx* ga = p.g[0] + (int64_t)tile * na;
    const cplx* gb = p.g[1] + (int64_t)tile * nb;
    for (int e = threadIdx.x; e < na; e += blockDim.x) gsm[e] = __ldg(ga + e);
    for (int e = threadIdx.x; e < nb; e += blockDim.x) gsm[na + e] = __ldg(gb + e);
    if (fh) {      // [P_a][2][WT] then [P_b][2][WT] behind the two g slices
        const cplx* fa = p.FH[0] + (int64_t)tile * 2 * na;
        const cplx* fb = p.FH[1] + (int64_t)tile * 2 * nb;
        cplx* dst = gsm + na + nb;
        for (int e = threadIdx.x; e < 2 * na; e += blockDim.x) dst[e] = __ldg(fa + e);
        for (int e = threadIdx.x; e < 2 * nb; e += blockDim.x) dst[2 * na + e] = __ldg(fb + e);
    }
    __syncthreads();
}

#define CF_CASE(KA_, KB_)                                                                              \
    case KA_ * 5 + KB_:                                                                                \
        if constexpr ((KA_ > KB_ ? KA_ : KB_) > KLO && (KA_ > KB_ ? KA_ : KB_) <= KHI)                  \
            run_bucket<KA_, KB_, MODE, FHS>(p, it, tile, slot, nslots, j, gsm, gpa, gpb, Wl, El, Hl);           \
        break;

// register class (KLO, KHI]: buckets whose larger level lies in that range (KLO = -1 admits (0,0)).
// Persistent per walker tile: CTA (worker, tile) stages g once and strides over the class's work items.
// GSM: the tile's g slices are staged in shared memory; false (windows wider than ~1800 pairs: they do not fit) reads them
// through L1/L2 and needs no dynamic shared memory at all (FHS implies GSM).
template <int MODE, int KLO, int KHI, int NTHR, int MINB, bool FHS, bool GSM = true>
__global__ void __launch_bounds__(NTHR, MINB) k_dets_cf(DetsParams p, const WorkItem* __restrict__ items, int n_items)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* gsm = reinterpret_cast<cplx*>(smem_raw);
    const int tile = blockIdx.y;
    const int j = threadIdx.x & (MSD_WT - 1);
    const int slot = threadIdx.x / MSD_WT, nslots = NTHR / MSD_WT;
    const cplx* gpa = gsm + j;
    const cplx* gpb = gsm + p.P[0] * MSD_WT + j;
    if (GSM) stage_g(p, tile, gsm, FHS);
    else { gpa = p.g[0] + (int64_t)tile * p.P[0] * MSD_WT + j; gpb = p.g[1] + (int64_t)tile * p.P[1] * MSD_WT + j; }
    cplx Wl = cmake(0.0, 0.0), El = cmake(0.0, 0.0), Hl = cmake(0.0, 0.0);
    for (int r = 0, ii; (ii = r * (int)gridDim.x + ((r & 1) ? (int)gridDim.x - 1 - (int)blockIdx.x : (int)blockIdx.x)),
                        r * (int)gridDim.x < n_items; r++) {
        if (ii >= n_items) continue;
        const WorkItem it = items[ii];
        switch (it.ka * 5 + it.kb) {
            CF_CASE(0, 0) CF_CASE(0, 1) CF_CASE(0, 2) CF_CASE(0, 3) CF_CASE(0, 4)
            CF_CASE(1, 0) CF_CASE(1, 1) CF_CASE(1, 2) CF_CASE(1, 3) CF_CASE(1, 4)
            CF_CASE(2, 0) CF_CASE(2, 1) CF_CASE(2, 2) CF_CASE(2, 3) CF_CASE(2, 4)
            CF_CASE(3, 0) CF_CASE(3, 1) CF_CASE(3, 2) CF_CASE(3, 3) CF_CASE(3, 4)
            CF_CASE(4, 0) CF_CASE(4, 1) CF_CASE(4, 2) CF_CASE(4, 3) CF_CASE(4, 4)
            default: break;
        }
    }
    flush_walker_sums(p, tile, Wl, El, Hl, MODE);
}

// ------------------------------------------------------------------------------------------------
// Force-bias mode of the closed-form levels: CI reduction by OWNER PULL (msd_internal.cuh PULL_*).  Nothing is scattered:
//   pass A  thread = (determinant, walker): R^a, R^b (levels <= 2: determinant only; levels 3, 4: determinant and adjugate by
//           the division-free closed forms, adjugate left UNSCALED in shared memory), W += c~ R^a R^b, and the two scale
//           factors c~ R^b (for alpha entries), c~ R^a (for beta entries) to shared memory;
//   pass B  lane group q (8 walkers) walks piece q of the chunk's entry list, which the setup sorted by pair index x and cut at
//           changes of x: the sum of an x-run stays in registers and is added to the CTA's C tile once, by its only owner.
// Replaces round 1's k_dets_c1 (products staged per round of 32-96 determinants, owner lists by x mod S read entry by entry
// with a shared-memory read-modify-write each: 2.0 ms at fe2s2, FP64 pipe 10-20 %).
// ------------------------------------------------------------------------------------------------
template <int K> __device__ __forceinline__ cplx det_only(const cplx (*M)[K > 0 ? K : 1])
{
    if constexpr (K == 0) return cmake(1.0, 0.0);
    else if constexpr (K == 1) return M[0][0];
    else return minor2(M[0][0], M[0][1], M[1][0], M[1][1]);
}

// byte `i` (compile-time after unrolling) of a table row held in registers as 32-bit words
template <int NWORD> __device__ __forceinline__ int row_byte(const uint32_t (&w)[NWORD], int i)
{
    return (int)((w[i >> 2] >> (8 * (i & 3))) & 255u);
}

// one spin of pass A: gather, determinant; levels >= 3 also leave the adjugate, element a*K+b = A[b][a], at
// stage[(a*K+b) * stride]  (stride = 8 x determinants of the chunk: consecutive threads -> consecutive 16-byte words)
template <int K, int OFF, int NWORD>
__device__ __forceinline__ cplx pull_spin(const uint32_t (&w)[NWORD], const cplx* g, int no, cplx* stage, int stride)
{
    constexpr int K1 = K > 0 ? K : 1;
    cplx M[K1][K1];
    int h[K1], pn[K1];
#pragma unroll
    for (int a = 0; a < K; a++) { h[a] = row_byte(w, OFF + a); pn[a] = row_byte(w, OFF + K + a) * no; }
#pragma unroll
    for (int a = 0; a < K; a++)
#pragma unroll
        for (int b = 0; b < K; b++) M[a][b] = g[(pn[b] + h[a]) * MSD_WT];
    if constexpr (K <= 2) return det_only<K>(M);
    else {
        cplx A[K1][K1];
        const cplx R = Closed<K>::det_adj(M, A);
#pragma unroll
        for (int a = 0; a < K; a++)
#pragma unroll
            for (int b = 0; b < K; b++) stage[(a * K + b) * stride] = A[b][a];
        return R;
    }
}

template <int KA, int KB>
__device__ __forceinline__ void pull_pass_a(const DetsParams& p, const WorkItem& it, int slot, int nslots, int j, const cplx* gA,
                                            const cplx* gB, cplx* sR, cplx* stage, cplx& Wl)
{
    constexpr int NB = 2 * KA + 2 * KB;
    constexpr int NWORD = (NB + 3) / 4 > 0 ? (NB + 3) / 4 : 1;
    constexpr int EA = KA >= 3 ? KA * KA : 0;
    const unsigned char* tab = p.tab + it.tab_off;
    const double* coef = p.coef + it.det_begin;
    const int stride = it.det_count * MSD_WT;
    for (int i = slot; i < it.det_count; i += nslots) {
        uint32_t w[NWORD];
        const uint32_t* rp = reinterpret_cast<const uint32_t*>(tab + (int64_t)i * it.rs);
#pragma unroll
        for (int t = 0; t < NWORD; t++) w[t] = (NB > 0) ? __ldg(rp + t) : 0u;
        const double cf = __ldg(coef + i);
        cplx* st = stage + i * MSD_WT + j;
        const cplx Ra = pull_spin<KA, 0>(w, gA, p.no[0], st, stride);
        const cplx Rb = pull_spin<KB, 2 * KA>(w, gB, p.no[1], st + EA * stride, stride);
        const cplx cRa = cscale(cf, Ra), cRb = cscale(cf, Rb);
        Wl = cfma(cRa, Rb, Wl);
        sR[(i * 2 + 0) * MSD_WT + j] = cRb;       // scale of the alpha entries
        sR[(i * 2 + 1) * MSD_WT + j] = cRa;       // scale of the beta entries
    }
}

__device__ __forceinline__ cplx flip(cplx v, uint32_t neg)       // neg = 0 or 1: integer sign flip, keeps the FP64 pipe free
{
    const long long m = (long long)neg << 63;
    return make_double2(__longlong_as_double(__double_as_longlong(v.x) ^ m), __longlong_as_double(__double_as_longlong(v.y) ^ m));
}

#define PULL_CASE(KA_, KB_)                                                                            \
    case KA_ * 5 + KB_:                                                                                \
        if constexpr ((KA_ > KB_ ? KA_ : KB_) > KLO && (KA_ > KB_ ? KA_ : KB_) <= KHI)                  \
            pull_pass_a<KA_, KB_>(p, it, slot, NTHR / MSD_WT, j, gA, gB, sR, stage, Wl);               \
        break;

// class (KLO, KHI] of the larger level; GS: the tile's g slices are staged in shared memory (else read through L1)
template <int NTHR, int KLO, int KHI, bool GS>
__global__ void __launch_bounds__(NTHR, 1) k_dets_pull(DetsParams p, const WorkItem* __restrict__ items, int n_items,
                                                       const unsigned short* __restrict__ pull_off,
                                                       const uint2* __restrict__ pull_ent, int pool_bytes)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int PT = p.P[0] + p.P[1];
    cplx* Csm = reinterpret_cast<cplx*>(smem_raw);                  // [(P_a + P_b)][WT]
    cplx* one = Csm + PT * MSD_WT;                                  // 16 walkers' worth of the constant 1.0 (level-1 entries)
    cplx* sR = one + 2 * MSD_WT;                                    // pool: [D][2][WT] scale factors, then the staged adjugates
    cplx* gsm = reinterpret_cast<cplx*>(reinterpret_cast<unsigned char*>(sR) + pool_bytes);     // [(P_a + P_b)][WT]   (GS)
    if (threadIdx.x < 2 * MSD_WT) one[threadIdx.x] = cmake(1.0, 0.0);
    const int tile = blockIdx.y;
    const int j = threadIdx.x & (MSD_WT - 1);
    const int slot = threadIdx.x / MSD_WT;
    const cplx* g0 = GS ? gsm : p.g[0] + (int64_t)tile * p.P[0] * MSD_WT;
    const cplx* g1 = GS ? gsm + p.P[0] * MSD_WT : p.g[1] + (int64_t)tile * p.P[1] * MSD_WT;
    const cplx* gA = g0 + j;
    const cplx* gB = g1 + j;
    if (GS) {
        const cplx* ga = p.g[0] + (int64_t)tile * p.P[0] * MSD_WT;
        const cplx* gb = p.g[1] + (int64_t)tile * p.P[1] * MSD_WT;
        for (int e = threadIdx.x; e < p.P[0] * MSD_WT; e += NTHR) gsm[e] = __ldg(ga + e);
        for (int e = threadIdx.x; e < p.P[1] * MSD_WT; e += NTHR) gsm[p.P[0] * MSD_WT + e] = __ldg(gb + e);
    }
    for (int e = threadIdx.x; e < PT * MSD_WT; e += NTHR) Csm[e] = cmake(0.0, 0.0);
    __syncthreads();
    cplx Wl = cmake(0.0, 0.0);
    for (int r0 = 0, ii; (ii = r0 * (int)gridDim.x + ((r0 & 1) ? (int)gridDim.x - 1 - (int)blockIdx.x : (int)blockIdx.x)),
                         r0 * (int)gridDim.x < n_items; r0++) {
        if (ii >= n_items) continue;
        const WorkItem it = items[ii];
        cplx* stage = sR + it.det_count * 2 * MSD_WT;               // [E_staged][det_count][WT]
        // this group's piece of the entry list; its first 8 entries are requested before pass A
        const uint2* ent = pull_ent + it.sched_off;
        const int t0 = __ldg(pull_off + it.pull_off + slot), t1 = __ldg(pull_off + it.pull_off + slot + 1);
        uint2 nxt = (t0 + j < t1) ? __ldg(ent + t0 + j) : make_uint2(0u, 0u);
        switch (it.ka * 5 + it.kb) {
            PULL_CASE(0, 0) PULL_CASE(0, 1) PULL_CASE(0, 2) PULL_CASE(0, 3) PULL_CASE(0, 4)
            PULL_CASE(1, 0) PULL_CASE(1, 1) PULL_CASE(1, 2) PULL_CASE(1, 3) PULL_CASE(1, 4)
            PULL_CASE(2, 0) PULL_CASE(2, 1) PULL_CASE(2, 2) PULL_CASE(2, 3) PULL_CASE(2, 4)
            PULL_CASE(3, 0) PULL_CASE(3, 1) PULL_CASE(3, 2) PULL_CASE(3, 3) PULL_CASE(3, 4)
            PULL_CASE(4, 0) PULL_CASE(4, 1) PULL_CASE(4, 2) PULL_CASE(4, 3) PULL_CASE(4, 4)
            default: break;
        }
        if (it.ka + it.kb == 0) continue;                           // the reference determinant: W only (uniform over the CTA)
        __syncthreads();
        // pass B: branch-free per entry -- value and scale factor are plain shared-memory reads at offsets the setup computed
        {
            const unsigned char* sm_j = smem_raw + j * sizeof(cplx);
            const unsigned char* sr_j = reinterpret_cast<const unsigned char*>(sR) + j * sizeof(cplx);
            cplx acc = cmake(0.0, 0.0);
            const unsigned gmask = 0xffu << (threadIdx.x & 24);     // the 8 lanes of this group
            for (int base = t0; base < t1; base += MSD_WT) {
                const uint2 mine = nxt;
                if (base + MSD_WT + j < t1) nxt = __ldg(ent + base + MSD_WT + j);
                const int n = t1 - base;
                // four entries at a time: their eight shared-memory reads are issued before any add to the C tile (the compiler
                // cannot move a load above the conditional store, but the C tile never aliases the operands)
#pragma unroll
                for (int i0 = 0; i0 < MSD_WT; i0 += 4) {
                    uint32_t w0[4];
                    cplx sv[4], vv[4];
#pragma unroll
                    for (int u = 0; u < 4; u++) {
                        w0[u] = __shfl_sync(gmask, mine.x, i0 + u, MSD_WT);
                        const uint32_t w1 = __shfl_sync(gmask, mine.y, i0 + u, MSD_WT);
                        const bool on = i0 + u < n;
                        sv[u] = *reinterpret_cast<const cplx*>(sr_j + (on ? (w0[u] & 0x3ffu) * 128u : 0u));
                        vv[u] = *reinterpret_cast<const cplx*>(sm_j + (on ? w1 : 0u));
                        if (!on) w0[u] = 0u;
                    }
#pragma unroll
                    for (int u = 0; u < 4; u++) {
                        if (i0 + u < n) acc = cfma(vv[u], flip(sv[u], (w0[u] >> 10) & 1u), acc);
                        if (w0[u] & (1u << 25)) {
                            cplx* cp = reinterpret_cast<cplx*>(smem_raw + ((w0[u] >> 11) & 0x3fffu) * 128u) + j;
                            cplx c0 = *cp; c0.x += acc.x; c0.y += acc.y; *cp = c0;
                            acc = cmake(0.0, 0.0);
                        }
                    }
                }
            }
        }
        __syncthreads();
    }
    // flush the CTA's C tile into the planar global accumulators
    for (int e = threadIdx.x; e < PT * MSD_WT; e += NTHR) {
        const cplx v = Csm[e];
        if (v.x == 0.0 && v.y == 0.0) continue;
        const int x = e / MSD_WT, jj = e - x * MSD_WT;
        const int sp = x >= p.P[0];
        const int xl = sp ? x - p.P[0] : x;
        double* C = p.C[sp] + (int64_t)tile * p.P[sp] * 2 * MSD_WT + jj;
        red_add_planar(C, xl, v);
    }
    flush_walker_sums(p, tile, Wl, cmake(0.0, 0.0), cmake(0.0, 0.0), 1);
}

// ------------------------------------------------------------------------------------------------
// generic levels (k >= 5 in at least one spin): one matrix per thread in shared memory, element e of
// thread t at sm[e * T + t] (consecutive lanes -> consecutive 16-byte words: conflict-free for any per-lane e).
// After a spin is evaluated its region holds A (entry e = b*k+a is A[b][a]) and the int region holds the pair
// index x(a,b) of the same entry.  Levels 5..8 run with compile-time K (unrolled gathers: K^2 / C(K,2) independent
// L2 loads in flight per thread); anything above 8 takes the runtime-k path.
// ------------------------------------------------------------------------------------------------
struct SmMat {
    cplx* base; int T;
    __device__ __forceinline__ cplx& at(int e) { return base[e * T]; }
};
typedef unsigned short xidx_t;      // a pair index x < n_o n_v <= 8192 (include/msd.h); 16 bits keep the per-thread footprint at 18 B per element
struct SmIdx {
    xidx_t* base; int T;
    __device__ __forceinline__ xidx_t& at(int e) { return base[e * T]; }
};

// in-place Gauss-Jordan inverse with partial pivoting; returns det (0 if an exactly zero pivot appears,
// in which case the matrix content is zeroed: adj and second cofactors are taken as 0 -- reading A11)
__device__ cplx gauss_jordan(SmMat m, int k)
{
    unsigned long long ipiv = 0ull;          // 4 bits per pivot row (k <= 16)
    cplx det = cmake(1.0, 0.0);
    bool sing = false;
    for (int j = 0; j < k; j++) {
        int p = j; double best = cabs2(m.at(j * k + j));
        for (int i = j + 1; i < k; i++) { double v = cabs2(m.at(i * k + j)); if (v > best) { best = v; p = i; } }
        ipiv |= (unsigned long long)p << (4 * j);
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
        int p = (int)((ipiv >> (4 * j)) & 15ull);
        if (p != j)
            for (int i = 0; i < k; i++) { cplx t = m.at(i * k + j); m.at(i * k + j) = m.at(i * k + p); m.at(i * k + p) = t; }
    }
    return det;
}

// the same elimination with compile-time K: the scaled pivot row lives in registers, so every update is one
// shared-memory load and one store
template <int K>
__device__ __forceinline__ cplx gauss_jordan_t(SmMat m)
{
    unsigned ipiv = 0u;                       // 4 bits per pivot row (K <= 8)
    cplx det = cmake(1.0, 0.0);
    bool sing = false;
    // K <= 6: pivot steps unrolled too (the c == j / i > j tests resolve at compile time: no selects in the update)
#pragma unroll (K <= 6 ? K : 1)
    for (int j = 0; j < K; j++) {
        int p = j; double best = cabs2(m.at(j * K + j));
#pragma unroll
        for (int i = 1; i < K; i++) {
            if (i > j) { double v = cabs2(m.at(i * K + j)); if (v > best) { best = v; p = i; } }
        }
        ipiv |= (unsigned)p << (4 * j);
        if (!(best > 0.0)) { sing = true; break; }
        cplx prow[K];
#pragma unroll
        for (int c = 0; c < K; c++) prow[c] = m.at(p * K + c);
        if (p != j) {
#pragma unroll
            for (int c = 0; c < K; c++) m.at(p * K + c) = m.at(j * K + c);
            det = cneg(det);
        }
        cplx pv = cmake(0.0, 0.0);
#pragma unroll
        for (int c = 0; c < K; c++) if (c == j) { pv = prow[c]; prow[c] = cmake(1.0, 0.0); }
        det = cmul(det, pv);
        const cplx r = cinv(pv);
#pragma unroll
        for (int c = 0; c < K; c++) { prow[c] = cmul(prow[c], r); m.at(j * K + c) = prow[c]; }
#pragma unroll
        for (int i = 0; i < K; i++) {
            if (i == j) continue;
            const cplx f = m.at(i * K + j);
#pragma unroll
            for (int c = 0; c < K; c++) {
                cplx v = m.at(i * K + c);
                if (c == j) v = cmake(0.0, 0.0);
                m.at(i * K + c) = cfms(f, prow[c], v);
            }
        }
    }
    if (sing) {
#pragma unroll
        for (int e = 0; e < K * K; e++) m.at(e) = cmake(0.0, 0.0);
        return cmake(0.0, 0.0);
    }
#pragma unroll 1
    for (int j = K - 1; j >= 0; j--) {
        const int p = (int)((ipiv >> (4 * j)) & 15u);
        if (p != j) {
#pragma unroll
            for (int i = 0; i < K; i++) { cplx t = m.at(i * K + j); m.at(i * K + j) = m.at(i * K + p); m.at(i * K + p) = t; }
        }
    }
    return det;
}

// Determinant only (overlap mode needs no adjugate): the forward half of the same elimination -- same pivots, same
// operation order as gauss_jordan / gauss_jordan_t on the rows below the pivot, hence the same value -- at a third of the
// shared-memory traffic.  0 for an exactly singular matrix.
__device__ cplx det_lu(SmMat m, int k)
{
    cplx det = cmake(1.0, 0.0);
    for (int j = 0; j < k; j++) {
        int p = j; double best = cabs2(m.at(j * k + j));
        for (int i = j + 1; i < k; i++) { double v = cabs2(m.at(i * k + j)); if (v > best) { best = v; p = i; } }
        if (!(best > 0.0)) return cmake(0.0, 0.0);
        if (p != j) {
            for (int c = j; c < k; c++) { cplx t = m.at(j * k + c); m.at(j * k + c) = m.at(p * k + c); m.at(p * k + c) = t; }
            det = cneg(det);
        }
        const cplx pv = m.at(j * k + j);
        det = cmul(det, pv);
        const cplx r = cinv(pv);
        for (int c = j + 1; c < k; c++) m.at(j * k + c) = cmul(m.at(j * k + c), r);
        for (int i = j + 1; i < k; i++) {
            const cplx f = m.at(i * k + j);
            for (int c = j + 1; c < k; c++) m.at(i * k + c) = cfms(f, m.at(j * k + c), m.at(i * k + c));
        }
    }
    return det;
}

template <int K>
__device__ __forceinline__ cplx det_lu_t(SmMat m)
{
    cplx det = cmake(1.0, 0.0);
    bool sing = false;
#pragma unroll (K <= 6 ? K : 1)
    for (int j = 0; j < K; j++) {
        int p = j; double best = cabs2(m.at(j * K + j));
#pragma unroll
        for (int i = 1; i < K; i++) {
            if (i > j) { double v = cabs2(m.at(i * K + j)); if (v > best) { best = v; p = i; } }
        }
        if (!(best > 0.0)) { sing = true; break; }
        cplx prow[K];                             // columns <= j are never read again
#pragma unroll
        for (int c = 0; c < K; c++) if (c >= j) prow[c] = m.at(p * K + c);
        if (p != j) {
#pragma unroll
            for (int c = 0; c < K; c++) if (c >= j) m.at(p * K + c) = m.at(j * K + c);
            det = cneg(det);
        }
        cplx pv = cmake(1.0, 0.0);
#pragma unroll
        for (int c = 0; c < K; c++) if (c == j) pv = prow[c];
        det = cmul(det, pv);
        const cplx r = cinv(pv);
#pragma unroll
        for (int c = 0; c < K; c++) if (c > j) prow[c] = cmul(prow[c], r);
#pragma unroll
        for (int i = 1; i < K; i++) {
            if (i <= j) continue;
            const cplx f = m.at(i * K + j);
#pragma unroll
            for (int c = 1; c < K; c++)
                if (c > j) m.at(i * K + c) = cfms(f, prow[c], m.at(i * K + c));
        }
    }
    return sing ? cmake(0.0, 0.0) : det;
}

// levels 1..4 inside the generic kernel (the other spin of a high-level bucket): closed forms in registers,
// A and x written to the thread's shared-memory regions
template <int K>
__device__ __forceinline__ cplx closed_to_smem(SmMat m, SmIdx xs, const unsigned char* hp, const cplx* __restrict__ g, int no,
                                               cplx* Ess, const cplx* __restrict__ Vss, unsigned P, int mode)
{
    int h[K], pn[K];
#pragma unroll
    for (int a = 0; a < K; a++) { h[a] = (int)hp[a]; pn[a] = (int)hp[K + a] * no; }
    cplx M[K][K], A[K][K];
#pragma unroll
    for (int a = 0; a < K; a++)
#pragma unroll
        for (int b = 0; b < K; b++) M[a][b] = __ldg(&g[(pn[b] + h[a]) * MSD_WT]);
    cplx R = Closed<K>::det_adj(M, A);
    if (mode == 0) { *Ess = cmake(0.0, 0.0); return R; }      // overlap: the determinant only (the adjugate is dead code)
#pragma unroll
    for (int a = 0; a < K; a++)
#pragma unroll
        for (int b = 0; b < K; b++) { m.at(b * K + a) = A[b][a]; xs.at(b * K + a) = pn[b] + h[a]; }
    cplx e = cmake(0.0, 0.0);
    if (mode >= 2 && K >= 2) {
#pragma unroll
        for (int a = 0; a < K; a++)
#pragma unroll
            for (int c = a + 1; c < K; c++)
#pragma unroll
                for (int b = 0; b < K; b++)
#pragma unroll
                    for (int d = b + 1; d < K; d++) {
                        cplx t = second_cofactor<K>(M, a, c, b, d);
                        e = cfma(t, __ldg(&Vss[((unsigned)(pn[b] + h[a]) * P + (unsigned)(pn[d] + h[c])) * MSD_WT]), e);
                    }
    }
    *Ess = e;
    return R;
}

// 5 x 5 Gauss-Jordan in registers (see k_dets_r5 below for the idea): WANT_INV leaves M^-1 in M, else only the determinant
template <bool WANT_INV>
__device__ __forceinline__ cplx gj5_reg(cplx (&M)[5][5])
{
    constexpr int K = 5;
    cplx det = cmake(1.0, 0.0);
    bool sing = false;
    unsigned swaps = 0u;                       // bit (4 j + i - j - 1): rows j and i were swapped in step j
#pragma unroll
    for (int j = 0; j < K; j++) {
#pragma unroll
        for (int i = j + 1; i < K; i++) {
            const bool sw = cabs2(M[i][j]) > cabs2(M[j][j]);
#pragma unroll
            for (int c = 0; c < K; c++) {
                if (!WANT_INV && c < j) continue;
                const cplx a = M[j][c], b = M[i][c];
                M[j][c] = sw ? b : a;
                M[i][c] = sw ? a : b;
            }
            if (sw) { det = cneg(det); swaps |= 1u << (4 * j + i - j - 1); }
        }
        const cplx pv = M[j][j];
        if (!(cabs2(pv) > 0.0)) sing = true;
        det = cmul(det, pv);
        const cplx r = sing ? cmake(0.0, 0.0) : cinv(pv);
        if (WANT_INV) M[j][j] = cmake(1.0, 0.0);
#pragma unroll
        for (int c = 0; c < K; c++) if (WANT_INV || c > j) M[j][c] = cmul(M[j][c], r);
#pragma unroll
        for (int i = 0; i < K; i++) {
            if (i == j || (!WANT_INV && i < j)) continue;
            const cplx f = M[i][j];
            if (WANT_INV) M[i][j] = cmake(0.0, 0.0);
#pragma unroll
            for (int c = 0; c < K; c++) if (WANT_INV || c > j) M[i][c] = cfms(f, M[j][c], M[i][c]);
        }
    }
    if (WANT_INV) {
#pragma unroll
        for (int j = K - 1; j >= 0; j--)
#pragma unroll
            for (int i = K - 1; i > j; i--) {
                const bool sw = (swaps >> (4 * j + i - j - 1)) & 1u;
#pragma unroll
                for (int rr = 0; rr < K; rr++) {
                    const cplx a = M[rr][j], b = M[rr][i];
                    M[rr][j] = sw ? b : a;
                    M[rr][i] = sw ? a : b;
                }
            }
        if (sing) {
#pragma unroll
            for (int a = 0; a < K; a++)
#pragma unroll
                for (int b = 0; b < K; b++) M[a][b] = cmake(0.0, 0.0);
        }
    }
    return sing ? cmake(0.0, 0.0) : det;
}

// levels 5..8 with compile-time K: gather, Gauss-Jordan, A = R M^-1, and the same-spin second-order sum
//   Ess = (1/R) sum_{a<c} sum_{b<d} (A[b][a] A[d][c] - A[b][c] A[d][a]) Vbar[x_ab][x_cd]        (Jacobi)
// with columns a and c of A in registers and the C(K,2) loads of one (a,c) pair independent of one another.
template <int K, int MODE, bool R5 = false>
__device__ __noinline__ cplx spin_big(cplx* mbase, xidx_t* xbase, int T, const unsigned char* hp, const cplx* __restrict__ g, int no,
                                      const cplx* __restrict__ Vss, unsigned P, cplx* Ess)
{
    SmMat m{mbase, T};
    SmIdx xs{xbase, T};
    int pn[K];
    unsigned long long hpack = 0ull;
#pragma unroll
    for (int a = 0; a < K; a++) { hpack |= (unsigned long long)hp[a] << (8 * a); pn[a] = (int)hp[K + a] * no; }
#pragma unroll
    for (int a = 0; a < K; a++) {
        const int ha = (int)((hpack >> (8 * a)) & 255ull);
        cplx row[K];
#pragma unroll
        for (int b = 0; b < K; b++) row[b] = __ldg(&g[(pn[b] + ha) * MSD_WT]);
#pragma unroll
        for (int b = 0; b < K; b++) { m.at(a * K + b) = row[b]; if (MODE != 0) xs.at(b * K + a) = pn[b] + ha; }
    }
    if (MODE == 0) { *Ess = cmake(0.0, 0.0); return det_lu_t<K>(m); }      // overlap: forward elimination only
    cplx R;
    if constexpr (R5 && K == 5) {
        // the kernel variant with a 255-register budget: inverse in registers, A written to shared memory once
        cplx Mr[5][5];
#pragma unroll
        for (int a = 0; a < 5; a++)
#pragma unroll
            for (int b = 0; b < 5; b++) Mr[a][b] = m.at(a * 5 + b);
        R = gj5_reg<true>(Mr);
#pragma unroll
        for (int a = 0; a < 5; a++)
#pragma unroll
            for (int b = 0; b < 5; b++) m.at(a * 5 + b) = cmul(R, Mr[a][b]);
    } else {
        R = gauss_jordan_t<K>(m);                 // m = M^-1 (or zeros)
#pragma unroll
        for (int e = 0; e < K * K; e++) m.at(e) = cmul(R, m.at(e));   // A = R M^-1, entry b*K+a = A[b][a]
    }
    *Ess = cmake(0.0, 0.0);
    if (M_ENERGY(MODE) && (R.x != 0.0 || R.y != 0.0)) {
        cplx e2[2] = {cmake(0.0, 0.0), cmake(0.0, 0.0)};      // two chains: the FMA latency is not on the critical path
#pragma unroll 1
        for (int a = 0; a < K - 1; a++) {
            const unsigned ha = (unsigned)((hpack >> (8 * a)) & 255ull);
            cplx ca[K];
#pragma unroll
            for (int b = 0; b < K; b++) ca[b] = m.at(b * K + a);
#pragma unroll 1
            for (int c = a + 1; c < K; c++) {
                const unsigned hc = (unsigned)((hpack >> (8 * c)) & 255ull);
                const cplx* vac = Vss + (ha * P + hc) * MSD_WT;       // x_ab P + x_cd = (pn_b P + pn_d) + (h_a P + h_c)
                cplx cc[K];
#pragma unroll
                for (int b = 0; b < K; b++) cc[b] = m.at(b * K + c);
#pragma unroll
                for (int b = 0; b < K; b++)
#pragma unroll
                    for (int d = b + 1; d < K; d++) {
                        const cplx v = __ldg(vac + ((unsigned)pn[b] * P + (unsigned)pn[d]) * MSD_WT);
                        cplx t = cmul(ca[b], cc[d]);
                        t = cfms(cc[b], ca[d], t);
                        e2[(b + d) & 1] = cfma(t, v, e2[(b + d) & 1]);
                    }
            }
        }
        *Ess = cmul(cadd(e2[0], e2[1]), cinv(R));
    }
    return R;
}

// any level, runtime k (levels above 8)
__device__ __noinline__ cplx spin_runtime(cplx* mbase, xidx_t* xbase, int T, int k, const unsigned char* hp,
                                          const cplx* __restrict__ g, int no, const cplx* __restrict__ Vss, unsigned P, int mode,
                                          cplx* Ess)
{
    SmMat m{mbase, T};
    SmIdx xs{xbase, T};
    for (int a = 0; a < k; a++)
        for (int b = 0; b < k; b++) {
            const int x = (int)hp[k + b] * no + (int)hp[a];
            m.at(a * k + b) = __ldg(&g[x * MSD_WT]);
            xs.at(b * k + a) = x;
        }
    *Ess = cmake(0.0, 0.0);
    if (mode == 0) return det_lu(m, k);
    cplx R = gauss_jordan(m, k);
    for (int e = 0; e < k * k; e++) m.at(e) = cmul(R, m.at(e));
    if (mode >= 2 && (R.x != 0.0 || R.y != 0.0)) {
        cplx e = cmake(0.0, 0.0);
        for (int a = 0; a < k; a++)
            for (int c = a + 1; c < k; c++)
                for (int b = 0; b < k; b++) {
                    const cplx Aba = m.at(b * k + a), Abc = m.at(b * k + c);
                    const unsigned xab = (unsigned)xs.at(b * k + a) * P;
#pragma unroll 4
                    for (int d = b + 1; d < k; d++) {
                        const cplx v = __ldg(&Vss[(xab + (unsigned)xs.at(d * k + c)) * MSD_WT]);
                        cplx t = cmul(Aba, m.at(d * k + c));
                        t = cfms(Abc, m.at(d * k + a), t);
                        e = cfma(t, v, e);
                    }
                }
        *Ess = cmul(e, cinv(R));
    }
    return R;
}

template <int MODE, bool R5 = false>
__device__ __forceinline__ cplx spin_any(cplx* mbase, xidx_t* xbase, int T, int k, const unsigned char* hp, const cplx* __restrict__ g,
                                         int no, const cplx* __restrict__ Vss, unsigned P, cplx* Ess)
{
    SmMat m{mbase, T};
    SmIdx xs{xbase, T};
    switch (k) {
        case 0: *Ess = cmake(0.0, 0.0); return cmake(1.0, 0.0);
        case 1: return closed_to_smem<1>(m, xs, hp, g, no, Ess, Vss, P, MODE);
        case 2: return closed_to_smem<2>(m, xs, hp, g, no, Ess, Vss, P, MODE);
        case 3: return closed_to_smem<3>(m, xs, hp, g, no, Ess, Vss, P, MODE);
        case 4: return closed_to_smem<4>(m, xs, hp, g, no, Ess, Vss, P, MODE);
        case 5: return spin_big<5, MODE, R5>(mbase, xbase, T, hp, g, no, Vss, P, Ess);
        case 6: return spin_big<6, MODE>(mbase, xbase, T, hp, g, no, Vss, P, Ess);
        case 7: return spin_big<7, MODE>(mbase, xbase, T, hp, g, no, Vss, P, Ess);
        case 8: return spin_big<8, MODE>(mbase, xbase, T, hp, g, no, Vss, P, Ess);
        default: return spin_runtime(mbase, xbase, T, k, hp, g, no, Vss, P, MODE, Ess);
    }
}

// opposite-spin second-order sum  sum_v As[v] sum_u Ab[u] Vab[x_u, x_v]:  the K^2 loads of the higher-level spin
// are unrolled (independent, four accumulators), the other spin's entries are a runtime loop
template <int K>
__device__ __noinline__ cplx opp_big(const cplx* mbig, const xidx_t* xbig, const cplx* msm, const xidx_t* xsm, int T, int ns,
                                     const cplx* __restrict__ V, unsigned sbig, unsigned ssm)
{
    cplx e = cmake(0.0, 0.0);
#pragma unroll 1
    for (int v = 0; v < ns; v++) {
        const cplx As = msm[v * T];
        const cplx* vp = V + (unsigned)xsm[v * T] * ssm * MSD_WT;
        cplx z[4];
#pragma unroll
        for (int t = 0; t < 4; t++) z[t] = cmake(0.0, 0.0);
#pragma unroll
        for (int u = 0; u < K * K; u++)
            z[u & 3] = cfma(mbig[u * T], __ldg(vp + (unsigned)xbig[u * T] * sbig * MSD_WT), z[u & 3]);
        e = cfma(As, cadd(cadd(z[0], z[1]), cadd(z[2], z[3])), e);
    }
    return e;
}

__device__ __noinline__ cplx opp_runtime(const cplx* mbig, const xidx_t* xbig, int nb, const cplx* msm, const xidx_t* xsm, int T, int ns,
                                         const cplx* __restrict__ V, unsigned sbig, unsigned ssm)
{
    cplx e = cmake(0.0, 0.0);
    for (int v = 0; v < ns; v++) {
        const cplx As = msm[v * T];
        const cplx* vp = V + (unsigned)xsm[v * T] * ssm * MSD_WT;
        cplx z = cmake(0.0, 0.0);
#pragma unroll 4
        for (int u = 0; u < nb; u++) z = cfma(mbig[u * T], __ldg(vp + (unsigned)xbig[u * T] * sbig * MSD_WT), z);
        e = cfma(As, z, e);
    }
    return e;
}

// Persistent per walker tile like k_dets_cf; shared memory per thread = (ka^2+kb^2) x (complex + int), bounded by the
// launch group's element count.
// R5: the variant for the groups whose high spin is at level 5 (ka^2 + kb^2 <= 34) in the energy modes: 255 registers, the 5 x 5
// inverse in registers (gj5_reg), the adjugate written to shared memory once for the second-order loops
template <int MODE, bool R5 = false>
__global__ void __launch_bounds__(128, R5 ? 2 : 3) k_dets_gen(DetsParams p, const WorkItem* __restrict__ items, int n_items)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* gsm = reinterpret_cast<cplx*>(smem_raw);
    const int tile = blockIdx.y;
    const int j = threadIdx.x & (MSD_WT - 1);
    const int slot = threadIdx.x / MSD_WT, nslots = blockDim.x / MSD_WT;
    const int T = blockDim.x;
    unsigned dyn_smem;
    asm("mov.u32 %0, %%dynamic_smem_size;" : "=r"(dyn_smem));
    const int elems_group = (int)(dyn_smem / ((sizeof(cplx) + sizeof(xidx_t)) * T));     // (complex + index) per element per thread
    const cplx* gA = p.g[0] + (int64_t)tile * p.P[0] * MSD_WT + j;      // L1/L2 resident (57 KB per tile)
    const cplx* gB = p.g[1] + (int64_t)tile * p.P[1] * MSD_WT + j;
    double* CA = p.C[0] + (int64_t)tile * p.P[0] * 2 * MSD_WT + j;
    double* CB = p.C[1] + (int64_t)tile * p.P[1] * 2 * MSD_WT + j;
    const cplx* VA = (M_ENERGY(MODE)) ? p.Vss[0] + (int64_t)tile * p.P[0] * p.P[0] * MSD_WT + j : nullptr;
    const cplx* VB = (M_ENERGY(MODE)) ? p.Vss[1] + (int64_t)tile * p.P[1] * p.P[1] * MSD_WT + j : nullptr;
    const cplx* VAB = (M_ENERGY(MODE)) ? p.Vab + (int64_t)tile * p.P[0] * p.P[1] * MSD_WT + j : nullptr;
    const cplx* FHA = (M_ENERGY(MODE)) ? p.FH[0] + (int64_t)tile * p.P[0] * 2 * MSD_WT + j : nullptr;
    const cplx* FHB = (M_ENERGY(MODE)) ? p.FH[1] + (int64_t)tile * p.P[1] * 2 * MSD_WT + j : nullptr;
    cplx Wl = cmake(0.0, 0.0), El = cmake(0.0, 0.0), Hl = cmake(0.0, 0.0);
    // snake order over rounds: items are sorted by descending cost, so alternate the direction to even out
    // work items are sized for 128-thread CTAs (msd_api.cu); a smaller CTA takes 1/split of an item at a time
    const int split = 128 / (int)blockDim.x, n_virt = n_items * split;
    for (int r = 0, iv; (iv = r * (int)gridDim.x + ((r & 1) ? (int)gridDim.x - 1 - (int)blockIdx.x : (int)blockIdx.x)),
                        r * (int)gridDim.x < n_virt; r++) {
        if (iv >= n_virt) continue;
        const int ii = iv / split, part = iv - ii * split;
        const WorkItem it = items[ii];
        const int ka = it.ka, kb = it.kb;
        const int na = ka * ka, nb = kb * kb;
        cplx* mA = gsm + threadIdx.x;
        cplx* mB = mA + na * T;
        // the int region starts at the LAUNCH GROUP's element bound, not at this item's na + nb: warps of a CTA are not
        // synchronised at item boundaries, so an item-dependent split would let one warp's indices alias another's matrix
        xidx_t* xA = reinterpret_cast<xidx_t*>(gsm + elems_group * T) + threadIdx.x;
        xidx_t* xB = xA + na * T;
        for (int i = part * nslots + slot; i < it.det_count; i += nslots * split) {
            const uint32_t* rp = reinterpret_cast<const uint32_t*>(p.tab + it.tab_off + (int64_t)i * it.rs);
            union { uint32_t w[MSD_MAX_LEVEL]; unsigned char b[4 * MSD_MAX_LEVEL]; } row;
            for (int t = 0; t < it.rs / 4; t++) row.w[t] = __ldg(rp + t);
            const double cf = __ldg(&p.coef[it.det_begin + i]);
            cplx EssA, EssB;
            const cplx Ra = spin_any<MODE, R5>(mA, xA, T, ka, row.b, gA, p.no[0], VA, (unsigned)p.P[0], &EssA);
            const cplx Rb = spin_any<MODE, R5>(mB, xB, T, kb, row.b + 2 * ka, gB, p.no[1], VB, (unsigned)p.P[1], &EssB);
            const cplx cRa = cscale(cf, Ra), cRb = cscale(cf, Rb);
            Wl = cfma(cRa, Rb, Wl);
            if (M_ENERGY(MODE)) {
                cplx e = cmake(0.0, 0.0);
                if (na > 0 && nb > 0) {
                    const bool abig = ka >= kb;
                    const cplx* mb_ = abig ? mA : mB; const xidx_t* xb_ = abig ? xA : xB;
                    const cplx* ms_ = abig ? mB : mA; const xidx_t* xs_ = abig ? xB : xA;
                    const unsigned sbig = abig ? (unsigned)p.P[1] : 1u, ssm = abig ? 1u : (unsigned)p.P[1];
                    const int ns = abig ? nb : na;
                    switch (abig ? ka : kb) {
                        case 5: e = opp_big<5>(mb_, xb_, ms_, xs_, T, ns, VAB, sbig, ssm); break;
                        case 6: e = opp_big<6>(mb_, xb_, ms_, xs_, T, ns, VAB, sbig, ssm); break;
                        case 7: e = opp_big<7>(mb_, xb_, ms_, xs_, T, ns, VAB, sbig, ssm); break;
                        case 8: e = opp_big<8>(mb_, xb_, ms_, xs_, T, ns, VAB, sbig, ssm); break;
                        default: e = opp_runtime(mb_, xb_, abig ? na : nb, ms_, xs_, T, ns, VAB, sbig, ssm); break;
                    }
                }
                cplx shA = cmake(0.0, 0.0), sfA = shA, shB = shA, sfB = shA;
#pragma unroll 4
                for (int u = 0; u < na; u++) {
                    const cplx* q = FHA + xA[u * T] * (2 * MSD_WT);
                    const cplx a_ = mA[u * T];
                    shA = cfma(a_, __ldg(q), shA);
                    sfA = cfma(a_, __ldg(q + MSD_WT), sfA);
                }
#pragma unroll 4
                for (int u = 0; u < nb; u++) {
                    const cplx* q = FHB + xB[u * T] * (2 * MSD_WT);
                    const cplx b_ = mB[u * T];
                    shB = cfma(b_, __ldg(q), shB);
                    sfB = cfma(b_, __ldg(q + MSD_WT), sfB);
                }
                e = cfma(Rb, cadd(EssA, sfA), e);
                e = cfma(Ra, cadd(EssB, sfB), e);
                El.x = fma(cf, e.x, El.x);
                El.y = fma(cf, e.y, El.y);
                cplx hsum = cmul(Rb, shA);
                hsum = cfma(Ra, shB, hsum);
                Hl.x = fma(cf, hsum.x, Hl.x);
                Hl.y = fma(cf, hsum.y, Hl.y);
            }
            if (M_SCATTER(MODE)) {
#pragma unroll 4
                for (int e = 0; e < na; e++) red_add_planar(CA, xA[e * T], cmul(cRb, mA[e * T]));
#pragma unroll 4
                for (int e = 0; e < nb; e++) red_add_planar(CB, xB[e * T], cmul(cRa, mB[e * T]));
            }
        }
    }
    flush_walker_sums(p, tile, Wl, El, Hl, MODE);
}

// ------------------------------------------------------------------------------------------------
// Level 5 against levels 0..3, overlap and force-bias modes: the whole 5 x 5 Gauss-Jordan inverse in REGISTERS.
// k_dets_gen keeps one matrix per thread in shared memory and is bound by that traffic (LSU 80 % busy in these groups);
// here pivoting is a compare-and-swap of whole rows and the column permutation is undone by compare-and-swaps in reverse
// order, so every index is a compile-time constant and nothing leaves the register file.  A kernel of its own because the
// 25 complex need a 255-register budget (inside k_dets_gen ptxas puts them in local memory: DESIGN.md section 11).
// Pivots are the column maxima, as in gauss_jordan_t; exactly singular matrices give R = 0, A = 0 (reading A11).
// ------------------------------------------------------------------------------------------------
// one bucket (KA, KB) with one spin at level 5 and the other at 0..3
template <int MODE, int KA, int KB>
__device__ __forceinline__ void r5_bucket(const DetsParams& p, const WorkItem& it, int slot, int nslots, const cplx* __restrict__ gA,
                                          const cplx* __restrict__ gB, double* CA, double* CB, cplx& Wl)
{
    constexpr int KS = KA == 5 ? KB : KA;               // the small spin's level
    constexpr int KS1 = KS > 0 ? KS : 1;
    constexpr bool BIG_A = KA == 5;
    const cplx* gbig = BIG_A ? gA : gB;
    const cplx* gsml = BIG_A ? gB : gA;
    const int nob = BIG_A ? p.no[0] : p.no[1], nos = BIG_A ? p.no[1] : p.no[0];
    double* Cbig = BIG_A ? CA : CB;
    double* Csml = BIG_A ? CB : CA;
    for (int i = slot; i < it.det_count; i += nslots) {
        const uint32_t* rp = reinterpret_cast<const uint32_t*>(p.tab + it.tab_off + (int64_t)i * it.rs);
        union { uint32_t w[4]; unsigned char b[16]; } row;        // 2 (KA + KB) <= 16 bytes
#pragma unroll
        for (int t = 0; t < 4; t++) row.w[t] = (t < (2 * (KA + KB) + 3) / 4) ? __ldg(rp + t) : 0u;
        const double cf = __ldg(&p.coef[it.det_begin + i]);
        const unsigned char* hb = row.b + (BIG_A ? 0 : 2 * KA);
        const unsigned char* hs = row.b + (BIG_A ? 2 * KA : 0);
        // small spin first (its adjugate is at most 9 complex)
        cplx As[KS1][KS1];
        int xs_h[KS1], xs_p[KS1];
        cplx Rs = cmake(1.0, 0.0);
        if (KS > 0) {
            cplx Ms[KS1][KS1];
#pragma unroll
            for (int a = 0; a < KS; a++) { xs_h[a] = (int)hs[a]; xs_p[a] = (int)hs[KS + a] * nos; }
#pragma unroll
            for (int a = 0; a < KS; a++)
#pragma unroll
                for (int b = 0; b < KS; b++) Ms[a][b] = __ldg(&gsml[(xs_p[b] + xs_h[a]) * MSD_WT]);
            Rs = Closed<KS>::det_adj(Ms, As);
        }
        int hh[5], pp[5];
#pragma unroll
        for (int a = 0; a < 5; a++) { hh[a] = (int)hb[a]; pp[a] = (int)hb[5 + a] * nob; }
        cplx M[5][5];
#pragma unroll
        for (int a = 0; a < 5; a++)
#pragma unroll
            for (int b = 0; b < 5; b++) M[a][b] = __ldg(&gbig[(pp[b] + hh[a]) * MSD_WT]);
        const cplx Rb = gj5_reg<MODE == 1>(M);           // M = M^-1 (force-bias mode)
        const cplx cRb = cscale(cf, Rb), cRs = cscale(cf, Rs);
        Wl = cfma(cRb, Rs, Wl);
        if (MODE == 1) {
            // C^big[x(a,b)] += c Rs A[b][a],  A = Rb M^-1  (entry [b][a] of the inverse belongs to pair (a, b))
            const cplx sc = cmul(cRs, Rb);
#pragma unroll
            for (int a = 0; a < 5; a++)
#pragma unroll
                for (int b = 0; b < 5; b++) red_add_planar(Cbig, pp[b] + hh[a], cmul(sc, M[b][a]));
            if (KS > 0) {
#pragma unroll
                for (int a = 0; a < KS; a++)
#pragma unroll
                    for (int b = 0; b < KS; b++) red_add_planar(Csml, xs_p[b] + xs_h[a], cmul(cRb, As[b][a]));
            }
        }
    }
}

#define R5_CASE(KA_, KB_) case KA_ * 8 + KB_: r5_bucket<MODE, KA_, KB_>(p, it, slot, nslots, gA, gB, CA, CB, Wl); break;

template <int MODE>
__global__ void __launch_bounds__(128, 2) k_dets_r5(DetsParams p, const WorkItem* __restrict__ items, int n_items)
{
    const int tile = blockIdx.y;
    const int j = threadIdx.x & (MSD_WT - 1);
    const int slot = threadIdx.x / MSD_WT, nslots = blockDim.x / MSD_WT;
    const cplx* gA = p.g[0] + (int64_t)tile * p.P[0] * MSD_WT + j;
    const cplx* gB = p.g[1] + (int64_t)tile * p.P[1] * MSD_WT + j;
    double* CA = p.C[0] + (int64_t)tile * p.P[0] * 2 * MSD_WT + j;
    double* CB = p.C[1] + (int64_t)tile * p.P[1] * 2 * MSD_WT + j;
    cplx Wl = cmake(0.0, 0.0);
    for (int r = 0, ii; (ii = r * (int)gridDim.x + ((r & 1) ? (int)gridDim.x - 1 - (int)blockIdx.x : (int)blockIdx.x)),
                        r * (int)gridDim.x < n_items; r++) {
        if (ii >= n_items) continue;
        const WorkItem it = items[ii];
        switch (it.ka * 8 + it.kb) {
            R5_CASE(5, 0) R5_CASE(5, 1) R5_CASE(5, 2) R5_CASE(5, 3)
            R5_CASE(0, 5) R5_CASE(1, 5) R5_CASE(2, 5) R5_CASE(3, 5)
            default: break;
        }
    }
    flush_walker_sums(p, tile, Wl, cmake(0.0, 0.0), cmake(0.0, 0.0), MODE);
}

// ------------------------------------------------------------------------------------------------
// very high levels (ka^2 + kb^2 > 100), cooperative form: a warp = ONE determinant x 8 walkers x 4 helper lanes
// (lane = helper * 8 + walker).  The four helpers of a (determinant, walker) share its matrices in shared memory
// (element e of walker j at mw[e * 8 + j]) and split every loop -- pivot search, row updates, the V gathers -- four ways.
// One matrix per THREAD (k_dets_gen) needs 2-4 KB of shared memory per thread at these levels, i.e. one or two warps per
// SM; here it is a quarter of that.  (At levels 5..8 the per-thread form with compile-time K is faster: measured.)
// Partial sums of the helpers meet in flush_walker_sums (which already adds lanes j, j+8, j+16, j+24).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ cplx shfl_c(cplx v, int src) {
    return make_double2(__shfl_sync(0xffffffffu, v.x, src), __shfl_sync(0xffffffffu, v.y, src));
}

// in-place inverse of the k x k matrix of every walker of the warp (partial pivoting); returns det, 0 for an exactly
// singular matrix (content zeroed: reading A11).  All four helpers of a walker return the same value.
__device__ __noinline__ cplx co_gauss_jordan(cplx* mw, int k, int hq)
{
    unsigned long long ipiv = 0ull;
    cplx det = cmake(1.0, 0.0);
    bool sing = false;
    for (int j0 = 0; j0 < k; j0++) {
        int p = j0; double best = -1.0;
        for (int i = j0 + hq; i < k; i += 4) { const double v = cabs2(mw[(i * k + j0) * 8]); if (v > best) { best = v; p = i; } }
#pragma unroll
        for (int o = 8; o <= 16; o <<= 1) {
            const double ob = __shfl_xor_sync(0xffffffffu, best, o);
            const int op = __shfl_xor_sync(0xffffffffu, p, o);
            if (ob > best || (ob == best && op < p)) { best = ob; p = op; }
        }
        ipiv |= (unsigned long long)p << (4 * j0);
        if (!(best > 0.0)) sing = true;
        if (p != j0) {
            for (int c = hq; c < k; c += 4) { const cplx t = mw[(j0 * k + c) * 8]; mw[(j0 * k + c) * 8] = mw[(p * k + c) * 8]; mw[(p * k + c) * 8] = t; }
            det = cneg(det);
        }
        __syncwarp();
        const cplx pv = mw[(j0 * k + j0) * 8];
        det = cmul(det, pv);
        const cplx r = sing ? cmake(0.0, 0.0) : cinv(pv);
        __syncwarp();
        for (int c = hq; c < k; c += 4) {
            const cplx v = (c == j0) ? cmake(1.0, 0.0) : mw[(j0 * k + c) * 8];
            mw[(j0 * k + c) * 8] = cmul(v, r);
        }
        __syncwarp();
        for (int i = hq; i < k; i += 4) {
            if (i == j0) continue;
            const cplx f = mw[(i * k + j0) * 8];
            for (int c = 0; c < k; c++) {
                const cplx v = (c == j0) ? cmake(0.0, 0.0) : mw[(i * k + c) * 8];
                mw[(i * k + c) * 8] = cfms(f, mw[(j0 * k + c) * 8], v);
            }
        }
        __syncwarp();
    }
    for (int j0 = k - 1; j0 >= 0; j0--) {
        const int p = (int)((ipiv >> (4 * j0)) & 15ull);
        if (p != j0)
            for (int i = hq; i < k; i += 4) { const cplx t = mw[(i * k + j0) * 8]; mw[(i * k + j0) * 8] = mw[(i * k + p) * 8]; mw[(i * k + p) * 8] = t; }
        __syncwarp();
    }
    if (sing) {
        for (int e = hq; e < k * k; e += 4) mw[e * 8] = cmake(0.0, 0.0);
        det = cmake(0.0, 0.0);
    }
    __syncwarp();
    return det;
}

// determinant only (overlap mode): the forward half of co_gauss_jordan -- same pivots, same operations on the rows below
// the pivot, hence the same value; rows j0+1.. are dealt to the four helpers
__device__ __noinline__ cplx co_det_lu(cplx* mw, int k, int hq)
{
    cplx det = cmake(1.0, 0.0);
    bool sing = false;
    for (int j0 = 0; j0 < k; j0++) {
        int p = j0; double best = -1.0;
        for (int i = j0 + hq; i < k; i += 4) { const double v = cabs2(mw[(i * k + j0) * 8]); if (v > best) { best = v; p = i; } }
#pragma unroll
        for (int o = 8; o <= 16; o <<= 1) {
            const double ob = __shfl_xor_sync(0xffffffffu, best, o);
            const int op = __shfl_xor_sync(0xffffffffu, p, o);
            if (ob > best || (ob == best && op < p)) { best = ob; p = op; }
        }
        if (!(best > 0.0)) sing = true;
        if (p != j0) {
            for (int c = j0 + hq; c < k; c += 4) { const cplx t = mw[(j0 * k + c) * 8]; mw[(j0 * k + c) * 8] = mw[(p * k + c) * 8]; mw[(p * k + c) * 8] = t; }
            det = cneg(det);
        }
        __syncwarp();
        const cplx pv = mw[(j0 * k + j0) * 8];
        det = cmul(det, pv);
        const cplx r = sing ? cmake(0.0, 0.0) : cinv(pv);
        __syncwarp();
        for (int c = j0 + 1 + hq; c < k; c += 4) mw[(j0 * k + c) * 8] = cmul(mw[(j0 * k + c) * 8], r);
        __syncwarp();
        for (int i = j0 + 1 + hq; i < k; i += 4) {
            const cplx f = mw[(i * k + j0) * 8];
            for (int c = j0 + 1; c < k; c++) mw[(i * k + c) * 8] = cfms(f, mw[(j0 * k + c) * 8], mw[(i * k + c) * 8]);
        }
        __syncwarp();
    }
    return sing ? cmake(0.0, 0.0) : det;
}

// one spin of the warp's determinant.  mw: this lane's walker column of the spin's matrix region; xw: the spin's pair
// indices (one copy per warp).  On exit mw holds A (entry b*k+a = A[b][a]), xw[b*k+a] = x(a,b); returns R (all helpers);
// *ess = this helper's share of the same-spin second-order sum.
template <int MODE>
__device__ __forceinline__ cplx co_spin(cplx* mw, xidx_t* xw, int k, const unsigned char* hp, const cplx* __restrict__ g, int no,
                                        const cplx* __restrict__ Vss, unsigned P, int hq, int j, cplx* ess)
{
    *ess = cmake(0.0, 0.0);
    if (k == 0) return cmake(1.0, 0.0);
    if (k <= MSD_CF_MAX) {          // closed forms by helper 0, result shared through shared memory
        cplx R = cmake(0.0, 0.0);
        if (hq == 0) {
            SmMat m{mw, 8};
            SmIdx xs{xw, 1};
            switch (k) {
                case 1: R = closed_to_smem<1>(m, xs, hp, g, no, ess, Vss, P, MODE); break;
                case 2: R = closed_to_smem<2>(m, xs, hp, g, no, ess, Vss, P, MODE); break;
                case 3: R = closed_to_smem<3>(m, xs, hp, g, no, ess, Vss, P, MODE); break;
                default: R = closed_to_smem<4>(m, xs, hp, g, no, ess, Vss, P, MODE); break;
            }
        }
        __syncwarp();
        return shfl_c(R, j);
    }
    const int lane = hq * 8 + j;
    for (int e = lane; e < k * k; e += 32) {      // pair indices, once per warp
        const int b = e / k, a = e - b * k;
        xw[e] = (xidx_t)((int)hp[k + b] * no + (int)hp[a]);
    }
    __syncwarp();
    for (int e = hq; e < k * k; e += 4) {         // M[a][b] = g[x(a,b)]; x(a,b) sits at xw[b*k+a]
        const int a = e / k, b = e - a * k;
        mw[e * 8] = __ldg(&g[xw[b * k + a] * MSD_WT]);
    }
    __syncwarp();
    if (MODE == 0) return co_det_lu(mw, k, hq);      // overlap: no adjugate
    const cplx R = co_gauss_jordan(mw, k, hq);
    for (int e = hq; e < k * k; e += 4) mw[e * 8] = cmul(R, mw[e * 8]);      // A = R M^-1
    __syncwarp();
    if (M_ENERGY(MODE) && (R.x != 0.0 || R.y != 0.0)) {
        // T[b,d;a,c] = (A[b][a] A[d][c] - A[b][c] A[d][a]) / R; helper hq takes the (a,c) pairs t = hq, hq+4, ... so that
        // the four helpers of a walker work on four different pairs in the same instruction (all lanes active; dealing
        // the pairs out by "skip unless t % 4 == hq" ran every pair with 8 of 32 lanes: profiles/r02_probes.md)
        cplx e = cmake(0.0, 0.0);
        const int npair = k * (k - 1) / 2;
        for (int t = hq; t < npair; t += 4) {
            int a = 0, rem = t;
            while (rem >= k - 1 - a) { rem -= k - 1 - a; a++; }
            const int c = a + 1 + rem;
            for (int b = 0; b < k - 1; b++) {
                const cplx Aba = mw[(b * k + a) * 8], Abc = mw[(b * k + c) * 8];
                const unsigned xab = (unsigned)xw[b * k + a] * P;
#pragma unroll 4
                for (int d = b + 1; d < k; d++) {
                    const cplx v = __ldg(&Vss[(xab + (unsigned)xw[d * k + c]) * MSD_WT]);
                    cplx tt = cmul(Aba, mw[(d * k + c) * 8]);
                    tt = cfms(Abc, mw[(d * k + a) * 8], tt);
                    e = cfma(tt, v, e);
                }
            }
        }
        *ess = cmul(e, cinv(R));
    }
    return R;
}

template <int MODE>
__global__ void __launch_bounds__(128, 4) k_dets_coop(DetsParams p, const WorkItem* __restrict__ items, int n_items, int elems)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tile = blockIdx.y;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int j = lane & 7, hq = lane >> 3;
    cplx* mwarp = reinterpret_cast<cplx*>(smem_raw) + (size_t)wid * elems * 8;            // [elems][8 walkers]
    xidx_t* xwarp = reinterpret_cast<xidx_t*>(reinterpret_cast<cplx*>(smem_raw) + (size_t)nwarps * elems * 8) + wid * elems;
    const cplx* gA = p.g[0] + (int64_t)tile * p.P[0] * MSD_WT + j;
    const cplx* gB = p.g[1] + (int64_t)tile * p.P[1] * MSD_WT + j;
    double* CA = p.C[0] + (int64_t)tile * p.P[0] * 2 * MSD_WT + j;
    double* CB = p.C[1] + (int64_t)tile * p.P[1] * 2 * MSD_WT + j;
    const cplx* VA = (M_ENERGY(MODE)) ? p.Vss[0] + (int64_t)tile * p.P[0] * p.P[0] * MSD_WT + j : nullptr;
    const cplx* VB = (M_ENERGY(MODE)) ? p.Vss[1] + (int64_t)tile * p.P[1] * p.P[1] * MSD_WT + j : nullptr;
    const cplx* VAB = (M_ENERGY(MODE)) ? p.Vab + (int64_t)tile * p.P[0] * p.P[1] * MSD_WT + j : nullptr;
    const cplx* FHA = (M_ENERGY(MODE)) ? p.FH[0] + (int64_t)tile * p.P[0] * 2 * MSD_WT + j : nullptr;
    const cplx* FHB = (M_ENERGY(MODE)) ? p.FH[1] + (int64_t)tile * p.P[1] * 2 * MSD_WT + j : nullptr;
    cplx Wl = cmake(0.0, 0.0), El = cmake(0.0, 0.0), Hl = cmake(0.0, 0.0);
    for (int r = 0, ii; (ii = r * (int)gridDim.x + ((r & 1) ? (int)gridDim.x - 1 - (int)blockIdx.x : (int)blockIdx.x)),
                        r * (int)gridDim.x < n_items; r++) {
        if (ii >= n_items) continue;
        const WorkItem it = items[ii];
        const int ka = it.ka, kb = it.kb;
        const int na = ka * ka, nb = kb * kb;
        cplx* mA = mwarp + j;
        cplx* mB = mA + na * 8;
        xidx_t* xA = xwarp;
        xidx_t* xB = xwarp + na;
        for (int i = wid; i < it.det_count; i += nwarps) {
            const uint32_t* rp = reinterpret_cast<const uint32_t*>(p.tab + it.tab_off + (int64_t)i * it.rs);
            union { uint32_t w[MSD_MAX_LEVEL]; unsigned char b[4 * MSD_MAX_LEVEL]; } row;
            for (int t = 0; t < it.rs / 4; t++) row.w[t] = __ldg(rp + t);
            const double cf = __ldg(&p.coef[it.det_begin + i]);
            cplx EssA, EssB;
            const cplx Ra = co_spin<MODE>(mA, xA, ka, row.b, gA, p.no[0], VA, (unsigned)p.P[0], hq, j, &EssA);
            const cplx Rb = co_spin<MODE>(mB, xB, kb, row.b + 2 * ka, gB, p.no[1], VB, (unsigned)p.P[1], hq, j, &EssB);
            __syncwarp();
            const cplx cRa = cscale(cf, Ra), cRb = cscale(cf, Rb);
            if (hq == 0) Wl = cfma(cRa, Rb, Wl);
            if (M_ENERGY(MODE)) {
                // this helper's share: opposite-spin entries u = hq, hq+4, ... of alpha; Hrot / F entries likewise
                cplx e = cmake(0.0, 0.0), shA = e, sfA = e, shB = e, sfB = e;
                for (int u = hq; u < na; u += 4) {
                    const cplx Au = mA[u * 8];
                    const int xu = xA[u];
                    const cplx* vrow = VAB + (unsigned)xu * (unsigned)p.P[1] * MSD_WT;
                    cplx z0 = cmake(0.0, 0.0), z1 = z0;       // eight independent loads in flight, two FMA chains
                    int v = 0;
                    for (; v + 8 <= nb; v += 8) {
                        cplx w[8];
#pragma unroll
                        for (int t = 0; t < 8; t++) w[t] = __ldg(&vrow[xB[v + t] * MSD_WT]);
#pragma unroll
                        for (int t = 0; t < 8; t += 2) { z0 = cfma(mB[(v + t) * 8], w[t], z0); z1 = cfma(mB[(v + t + 1) * 8], w[t + 1], z1); }
                    }
                    for (; v < nb; v++) z0 = cfma(mB[v * 8], __ldg(&vrow[xB[v] * MSD_WT]), z0);
                    e = cfma(Au, cadd(z0, z1), e);
                    const cplx* q = FHA + xu * (2 * MSD_WT);
                    shA = cfma(Au, __ldg(q), shA);
                    sfA = cfma(Au, __ldg(q + MSD_WT), sfA);
                }
                for (int v = hq; v < nb; v += 4) {
                    const cplx Bv = mB[v * 8];
                    const cplx* q = FHB + xB[v] * (2 * MSD_WT);
                    shB = cfma(Bv, __ldg(q), shB);
                    sfB = cfma(Bv, __ldg(q + MSD_WT), sfB);
                }
                e = cfma(Rb, cadd(EssA, sfA), e);
                e = cfma(Ra, cadd(EssB, sfB), e);
                El.x = fma(cf, e.x, El.x);
                El.y = fma(cf, e.y, El.y);
                cplx hsum = cmul(Rb, shA);
                hsum = cfma(Ra, shB, hsum);
                Hl.x = fma(cf, hsum.x, Hl.x);
                Hl.y = fma(cf, hsum.y, Hl.y);
            }
            if (M_SCATTER(MODE)) {
                for (int u = hq; u < na; u += 4) red_add_planar(CA, xA[u], cmul(cRb, mA[u * 8]));
                for (int v = hq; v < nb; v += 4) red_add_planar(CB, xB[v], cmul(cRa, mB[v * 8]));
            }
            __syncwarp();       // the next determinant overwrites the warp's matrices
        }
    }
    flush_walker_sums(p, tile, Wl, El, Hl, MODE);
}

// ------------------------------------------------------------------------------------------------
// Antisymmetrised same-spin tensor, in place: Vbar[x_ab][x_cd] = V[x_ab][x_cd] - V[x_ad][x_cb] on the entries
// (h_a < h_c, p_b < p_d) -- the only ones the same-spin sum reads (holes and particles of a determinant ascend).
// V[x_ad][x_cb] is read through the symmetry V[x][y] = V[y][x] as V[(p_b,h_c)][(p_d,h_a)], an entry no thread writes.
// ------------------------------------------------------------------------------------------------
__global__ void k_vbar(cplx* __restrict__ V, int no, int nv, int64_t nt)
{
    const int nhh = no * (no - 1) / 2, npp = nv * (nv - 1) / 2;
    const int64_t P = (int64_t)no * nv;
    const int64_t total = nt * npp * nhh * MSD_WT;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int j = (int)(idx % MSD_WT);
        int64_t t = idx / MSD_WT;
        int hh = (int)(t % nhh); t /= nhh;
        int pp = (int)(t % npp);
        const int64_t tile = t / npp;
        int ha = 0; while (hh >= no - 1 - ha) { hh -= no - 1 - ha; ha++; }
        const int hc = ha + 1 + hh;
        int pb = 0; while (pp >= nv - 1 - pb) { pp -= nv - 1 - pb; pb++; }
        const int pd = pb + 1 + pp;
        cplx* Vt = V + tile * P * P * MSD_WT + j;
        const int64_t x1 = (int64_t)pb * no + ha, y1 = (int64_t)pd * no + hc;
        const int64_t x2 = (int64_t)pb * no + hc, y2 = (int64_t)pd * no + ha;
        const cplx u1 = Vt[(x1 * P + y1) * MSD_WT], u2 = Vt[(x2 * P + y2) * MSD_WT];
        Vt[(x1 * P + y1) * MSD_WT] = csub(u1, u2);
    }
}

// Hrot and F ([n_w][P] each) interleaved per pair index with the walker fastest: FH[tile][x][0][j] = Hrot, [1][j] = F
__global__ void k_fh_tile(const cplx* __restrict__ Hrot, const cplx* __restrict__ F, cplx* __restrict__ FH, int P, int64_t nw,
                          int64_t nt)
{
    const int64_t total = nt * P * MSD_WT;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int j = (int)(idx % MSD_WT);
        const int64_t t = idx / MSD_WT;
        const int x = (int)(t % P);
        const int64_t tile = t / P, w = tile * MSD_WT + j;
        const cplx zero = cmake(0.0, 0.0);
        cplx* dst = FH + ((tile * P + x) * 2) * MSD_WT + j;
        dst[0] = (w < nw) ? Hrot[w * P + x] : zero;
        dst[MSD_WT] = (w < nw) ? F[w * P + x] : zero;
    }
}

// ------------------------------------------------------------------------------------------------
template <class K>
static cudaError_t launch_persistent(msd_ctx* c, K kernel, int nthr, size_t smem, int n_sm, const DetsParams& p,
                                     const WorkItem* items, int n_items, int ntiles, cudaStream_t st, int vsplit = 1)
{
    if (n_items == 0) return cudaSuccess;
    int occ = 1;
    cudaError_t e = func_config(c, (const void*)kernel, nthr, smem, &occ);
    if (e != cudaSuccess) return e;
    // about two walker tiles resident at a time (their V slices stay in L2), every SM full
    const int n_units = n_items * vsplit;      // k_dets_gen with CTAs below 128 threads works on 1/vsplit of an item at a time
    int workers = (n_sm * occ + 1) / 2;
    if (workers > n_units) workers = n_units;
    if (ntiles == 1) workers = n_units < n_sm * occ ? n_units : n_sm * occ;
    dim3 grid(workers, ntiles);
    kernel<<<grid, nthr, smem, st>>>(p, items, n_items);
    return cudaGetLastError();
}

// closed-form buckets of the force-bias mode by owner pull: one launch per class (larger level <= 3: 512 threads, == 4: 256)
template <int NTHR, int KLO, int KHI>
static cudaError_t launch_pull_class(msd_ctx* c, const DetsParams& p, int ntiles, int i0, int i1, cudaStream_t st)
{
    const int n_items = i1 - i0;
    if (n_items <= 0) return cudaSuccess;
    const size_t tile_bytes = (size_t)(p.P[0] + p.P[1]) * MSD_WT * sizeof(cplx);
    const size_t smem = tile_bytes + 256 + c->pull_pool + (c->pull_gs ? tile_bytes : 0);
    const void* kern = c->pull_gs ? (const void*)k_dets_pull<NTHR, KLO, KHI, true> : (const void*)k_dets_pull<NTHR, KLO, KHI, false>;
    cudaError_t e = func_config(c, kern, NTHR, smem, nullptr);
    if (e != cudaSuccess) return e;
    // one CTA per SM, all resident at once: workers x tiles <= waves x SMs
    const int waves = (ntiles + c->n_sm - 1) / c->n_sm;
    int workers = std::max(1, waves * c->n_sm / ntiles);
    workers = std::min(workers, n_items);
    if (c->pull_gs)
        k_dets_pull<NTHR, KLO, KHI, true><<<dim3(workers, ntiles), NTHR, smem, st>>>(p, c->d_items_pull + i0, n_items, c->d_pull_off,
                                                                                     c->d_pull_ent, (int)c->pull_pool);
    else
        k_dets_pull<NTHR, KLO, KHI, false><<<dim3(workers, ntiles), NTHR, smem, st>>>(p, c->d_items_pull + i0, n_items, c->d_pull_off,
                                                                                      c->d_pull_ent, (int)c->pull_pool);
    c->launches++;
    return cudaGetLastError();
}

template <int MODE>
static cudaError_t launch_mode(msd_ctx* c, const DetsParams& p, int ntiles, cudaStream_t st)
{
    const size_t gbytes = (size_t)(p.P[0] + p.P[1]) * MSD_WT * sizeof(cplx);
    // test hook (msd_set_option MSD_OPT_NO_SMEM_TILES): take the paths used when a walker tile's C / Hrot / F / g do not fit
    // in shared memory (RED scatter for the force bias, operands through L1), which no BASELINE config needs
    const bool no_tiles = c->no_smem_tiles >= 1;
    const bool gsm_ok = gbytes <= 200 * 1024 && c->no_smem_tiles < 2;
    // The launches below are independent (they only meet in the RED accumulators), so they are forked over the
    // context's side streams: the small high-level groups no longer serialise their tails behind one another.
    Fork f(c, st);
    int li = 0;
    // generic kernel first (longest per-item latency): one launch per shared-memory group, highest levels first
    for (size_t gi = c->gen_group_begin.size() - 1; gi-- > 0;) {
        const int i0 = c->gen_group_begin[gi], i1 = c->gen_group_begin[gi + 1];
        if (i1 == i0) continue;
        if (c->gen_group_elems[gi] > (MODE >= 2 ? c->coop_min_elems : c->coop_min_elems_fb)) {   // measured crossover (MSD_OPT_COOP_MIN_ELEMS)
            const int elems = c->gen_group_elems[gi];
            const size_t smem = (size_t)4 * elems * (8 * sizeof(cplx) + sizeof(xidx_t));
            auto kern = k_dets_coop<MODE>;
            int occ = 1;
            cudaError_t e = func_config(c, (const void*)kern, 128, smem, &occ);
            if (e != cudaSuccess) { f.join(); return e; }
            int workers = std::min(i1 - i0, (c->n_sm * occ + 1) / 2);
            if (ntiles == 1) workers = std::min(i1 - i0, c->n_sm * occ);
            kern<<<dim3(workers, ntiles), 128, smem, f.stream(li++)>>>(p, c->d_items_gen + i0, i1 - i0, elems);
            e = cudaGetLastError();
            if (e != cudaSuccess) { f.join(); return e; }
            c->launches++;
            continue;
        }
        // groups 0 and 1 (ka^2 + kb^2 <= 34) hold exactly the buckets with one spin at level 5 and the other at 0..3:
        // overlap and force-bias modes take the register-resident kernel
        if (MODE <= 1 && gi <= 1 && c->gen_group_elems[gi] <= 34) {
            cudaError_t e = launch_persistent(c, k_dets_r5<(MODE <= 1 ? MODE : 0)>, 128, 0, c->n_sm, p, c->d_items_gen + i0, i1 - i0, ntiles,
                                              f.stream(li++));
            if (e != cudaSuccess) { f.join(); return e; }
            c->launches++;
            continue;
        }
        // CTA size: 128 threads unless the group does not fit.  (Smaller CTAs would leave more warps resident -- shared
        // memory per thread is fixed by the group -- but measured slower: the extra shared memory comes out of the L1 that
        // holds the walker tile's g / Hrot / F slices.  profiles/r02_probes.md)
        const size_t per_thread = (size_t)c->gen_group_elems[gi] * (sizeof(cplx) + sizeof(xidx_t));
        int nthr = 128;
        while (nthr > 32 && per_thread * nthr > 200 * 1024) nthr -= 32;
        size_t smem = per_thread * nthr;
        const bool r5 = MODE >= 2 && gi <= 1 && c->gen_group_elems[gi] <= 34 && nthr == 128;
        cudaError_t e = r5 ? launch_persistent(c, k_dets_gen<MODE, (MODE >= 2)>, nthr, smem, c->n_sm, p, c->d_items_gen + i0, i1 - i0, ntiles,
                                               f.stream(li++), 1)
                           : launch_persistent(c, k_dets_gen<MODE>, nthr, smem, c->n_sm, p, c->d_items_gen + i0, i1 - i0, ntiles,
                                               f.stream(li++), 128 / nthr);
        if (e != cudaSuccess) { f.join(); return e; }
        c->launches++;
    }
    // force bias, closed-form levels: owner-pull kernel (one launch for all buckets) unless the tile does not fit
    bool cf_done = false;
    if constexpr (MODE == 1) {
        if (!no_tiles && c->pull_pool) {
            cudaError_t e = launch_pull_class<256, 3, 4>(c, p, ntiles, c->pull_class_begin[1], c->pull_class_begin[2], f.stream(li++));
            if (e == cudaSuccess)
                e = launch_pull_class<512, -1, 3>(c, p, ntiles, c->pull_class_begin[0], c->pull_class_begin[1], f.stream(li++));
            if (e != cudaSuccess) { f.join(); return e; }
            cf_done = true;
        }
    }
    // closed-form kernel: three register classes, items sorted by class on the host (msd_api.cu)
    for (int cl = 2; cl >= 0 && !cf_done; cl--) {
        const int i0 = c->cf_class_begin[cl], i1 = c->cf_class_begin[cl + 1];
        if (i1 == i0) continue;
        cudaError_t e;
        cudaStream_t s = f.stream(li++);
        // energy mode: one large CTA per SM that also holds Hrot / F of the tile in shared memory (same warps per SM as
        // the 2-3 smaller CTAs of the other modes); falls back to global Hrot / F when the tile does not fit
        bool fhs = false;
        if constexpr (MODE >= 2) {
            fhs = 3 * gbytes <= 200 * 1024 && !no_tiles;
            if (!fhs) {}
            else if (cl == 0) e = launch_persistent(c, k_dets_cf<MODE, -1, 2, 768, 1, true>, 768, 3 * gbytes, c->n_sm, p, c->d_items_cf + i0, i1 - i0, ntiles, s);
            else if (cl == 1) e = launch_persistent(c, k_dets_cf<MODE, 2, 3, 512, 1, true>, 512, 3 * gbytes, c->n_sm, p, c->d_items_cf + i0, i1 - i0, ntiles, s);
            else e = launch_persistent(c, k_dets_cf<MODE, 3, 4, 256, 1, true>, 256, 3 * gbytes, c->n_sm, p, c->d_items_cf + i0, i1 - i0, ntiles, s);
        }
        if (!fhs && gsm_ok) {
            if (cl == 0) e = launch_persistent(c, k_dets_cf<MODE, -1, 2, 256, 3, false>, 256, gbytes, c->n_sm, p, c->d_items_cf + i0, i1 - i0, ntiles, s);
            else if (cl == 1) e = launch_persistent(c, k_dets_cf<MODE, 2, 3, 256, 2, false>, 256, gbytes, c->n_sm, p, c->d_items_cf + i0, i1 - i0, ntiles, s);
            else e = launch_persistent(c, k_dets_cf<MODE, 3, 4, 128, 2, false>, 128, gbytes, c->n_sm, p, c->d_items_cf + i0, i1 - i0, ntiles, s);
        } else if (!fhs) {      // g through L1/L2 as well: no dynamic shared memory
            if (cl == 0) e = launch_persistent(c, k_dets_cf<MODE, -1, 2, 256, 3, false, false>, 256, 0, c->n_sm, p, c->d_items_cf + i0, i1 - i0, ntiles, s);
            else if (cl == 1) e = launch_persistent(c, k_dets_cf<MODE, 2, 3, 256, 2, false, false>, 256, 0, c->n_sm, p, c->d_items_cf + i0, i1 - i0, ntiles, s);
            else e = launch_persistent(c, k_dets_cf<MODE, 3, 4, 128, 2, false, false>, 128, 0, c->n_sm, p, c->d_items_cf + i0, i1 - i0, ntiles, s);
        }
        if (e != cudaSuccess) { f.join(); return e; }
        c->launches++;
    }
    cudaError_t e = f.join();
    return e != cudaSuccess ? e : f.err;
}

cudaError_t launch_dets(msd_ctx* c, int mode, int64_t nw, Workspace& ws, cudaStream_t st)
{
    DetsParams p;
    p.tab = c->d_tab; p.coef = c->d_coef;
    for (int s = 0; s < 2; s++) {
        p.g[s] = ws.g[s]; p.C[s] = ws.C[s]; p.Vss[s] = ws.Vss[s];
        p.no[s] = c->sp[s].n_o; p.P[s] = c->sp[s].P;
    }
    p.Vab = ws.Vab; p.Wacc = ws.Wacc; p.E2nd = ws.E2nd; p.E1nd = ws.E1nd;
    p.FH[0] = ws.FH[0]; p.FH[1] = ws.FH[1];
    int ntiles = (int)((nw + MSD_WT - 1) / MSD_WT);
    if (mode >= 2) {
        for (int s = 0; s < 2; s++) {
            const auto& sp = c->sp[s];
            if (sp.kmax < 2 || sp.n_o < 2 || sp.n_v < 2) continue;
            const int64_t total = (int64_t)ntiles * (sp.n_o * (sp.n_o - 1) / 2) * (sp.n_v * (sp.n_v - 1) / 2) * MSD_WT;
            const int blocks = (int)std::min<int64_t>((total + 255) / 256, (int64_t)c->n_sm * 16);
            k_vbar<<<blocks, 256, 0, st>>>(ws.Vss[s], sp.n_o, sp.n_v, ntiles);
            cudaError_t e = cudaGetLastError();
            if (e != cudaSuccess) return e;
            c->launches++;
        }
        for (int s = 0; s < 2; s++) {
            const auto& sp = c->sp[s];
            if (sp.P == 0) continue;
            const int64_t total = (int64_t)ntiles * sp.P * MSD_WT;
            k_fh_tile<<<(int)std::min<int64_t>((total + 255) / 256, (int64_t)c->n_sm * 8), 256, 0, st>>>(
                ws.Hrot[s], ws.F[s], ws.FH[s], sp.P, nw, ntiles);
            cudaError_t e = cudaGetLastError();
            if (e != cudaSuccess) return e;
            c->launches++;
        }
    }
    if (mode == 0) return launch_mode<0>(c, p, ntiles, st);
    if (mode == 1) return launch_mode<1>(c, p, ntiles, st);
    if (mode == 2) return launch_mode<2>(c, p, ntiles, st);
    return launch_mode<3>(c, p, ntiles, st);
}

// S5 Green's function rows, S7 dense energy intermediates (all but the two big GEMMs, which are in gemm.cu),
// S9 assembly.  Wick steps W5-W10 of DESIGN.md "The algorithm"; Eq. 7, Eq. 14, L98.
#include "msd_internal.cuh"

__device__ __forceinline__ double nan_d() { return __longlong_as_double(0x7ff8000000000000LL); }

// block-wide sum of a complex; result valid in thread 0
__device__ __forceinline__ cplx block_sum(cplx v)
{
    __shared__ double sred[2][32];
    for (int o = 16; o > 0; o >>= 1) {
        v.x += __shfl_down_sync(0xffffffffu, v.x, o);
        v.y += __shfl_down_sync(0xffffffffu, v.y, o);
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    __syncthreads();
    if (lane == 0) { sred[0][wid] = v.x; sred[1][wid] = v.y; }
    __syncthreads();
    if (wid == 0) {
        v.x = lane < nw ? sred[0][lane] : 0.0;
        v.y = lane < nw ? sred[1][lane] : 0.0;
        for (int o = 16; o > 0; o >>= 1) {
            v.x += __shfl_down_sync(0xffffffffu, v.x, o);
            v.y += __shfl_down_sync(0xffffffffu, v.y, o);
        }
    }
    return v;
}

// ------------------------------------------------------------------------------------------------
// S5: G^s = G0 + (1/W) Q0 C G0 restricted to its non-zero rows occ_ref U act_virt  (W5)
//   rows l < n      : G[occ_ref[l]][q] = Theta[q][l] - sum_h U[l][h] Theta[q][pos(h)],  U = Theta_v^T D
//   rows n + r'     : G[act_v[r']][q]  = sum_h D[r'][h] Theta[q][pos(h)],               D = C / W
// written planar (re row, im row) as the B operand of the force-bias GEMM; optionally scattered into the
// full N x N matrix (msd_greens).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_green_rows(int N, int ldN, SpinDev sa, SpinDev sb, int64_t nw, const cplx* __restrict__ theta_a,
             const cplx* __restrict__ theta_b, const double* __restrict__ C_a, const double* __restrict__ C_b,
             const cplx* __restrict__ Wacc, double* Gp_a, double* Gp_b, cplx* Gfull, int* wflags)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int s = blockIdx.y;
    const int64_t w = blockIdx.x;
    const SpinDev sp = s ? sb : sa;
    const int n = sp.n, no = sp.n_o, nv = sp.n_v;
    const cplx* theta = (s ? theta_b : theta_a) + w * (int64_t)N * n;
    const double* C = (s ? C_b : C_a) + (w / MSD_WT) * (int64_t)sp.P * 2 * MSD_WT + (w % MSD_WT);
    double* Gp = (s ? Gp_b : Gp_a);
    cplx* D = reinterpret_cast<cplx*>(smem_raw);     // [nv][no]
    cplx* U = D + nv * no;                            // [n][no]
    const int tid = threadIdx.x, nt = blockDim.x;
    const cplx W = Wacc[w];
    const bool bad = (W.x == 0.0 && W.y == 0.0) || (wflags[w] & 1);
    if (tid == 0 && s == 0 && (W.x == 0.0 && W.y == 0.0)) atomicOr(&wflags[w], 2);
    const cplx Winv = bad ? cmake(nan_d(), nan_d()) : cinv(W);
    for (int x = tid; x < nv * no; x += nt) D[x] = cmul(load_planar(C, x), Winv);
    __syncthreads();
    for (int e = tid; e < n * no; e += nt) {
        int l = e / no, h = e - l * no;
        cplx acc = cmake(0.0, 0.0);
        for (int r = 0; r < nv; r++) acc = cfma(theta[(int64_t)sp.act_v[r] * n + l], D[r * no + h], acc);
        U[e] = acc;
    }
    __syncthreads();
    const int nr = sp.n_r;
    const int64_t ldk = (int64_t)nr * ldN;
    double* gre = Gp ? Gp + (w * 2) * ldk : nullptr;
    double* gim = Gp ? gre + ldk : nullptr;
    cplx* Gf = Gfull ? Gfull + (w * 2 + s) * (int64_t)N * N : nullptr;
    for (int e = tid; e < nr * ldN; e += nt) {
        int r = e / ldN, q = e - r * ldN;
        cplx acc = cmake(0.0, 0.0);
        if (q < N) {
            const cplx* th = theta + (int64_t)q * n;
            if (r < n) {
                acc = th[r];
                for (int h = 0; h < no; h++) acc = cfms(U[r * no + h], th[sp.pos_o[h]], acc);
            } else {
                const cplx* d = D + (r - n) * no;
                for (int h = 0; h < no; h++) acc = cfma(d[h], th[sp.pos_o[h]], acc);
            }
            if (Gf) {
                int p = (r < n) ? sp.occ_ref[r] : sp.act_v[r - n];
                Gf[(int64_t)p * N + q] = acc;
            }
        }
        if (gre) { gre[e] = acc.x; gim[e] = acc.y; }
    }
}

cudaError_t launch_green_rows(msd_ctx* c, int64_t nw, Workspace& ws, cplx* Gfull, cudaStream_t st)
{
    if (nw == 0) return cudaSuccess;
    int ldN = c->N + (c->N & 1);
    size_t smem = 0;
    for (int s = 0; s < 2; s++) {
        size_t v = ((size_t)c->sp[s].n_v * c->sp[s].n_o + (size_t)c->sp[s].n * c->sp[s].n_o + 1) * sizeof(cplx);
        if (v > smem) smem = v;
    }
    cudaError_t e = func_config(c, (const void*)k_green_rows, 256, smem, nullptr);
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)nw, 2);
    k_green_rows<<<grid, 256, smem, st>>>(c->N, ldN, c->dev(0), c->dev(1), nw, ws.theta[0], ws.theta[1], ws.C[0],
                                          ws.C[1], ws.Wacc, ws.Gp[0], ws.Gp[1], Gfull, ws.wflags);
    c->launches++;
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// S7: from Lam = L_sub Theta (rows (g, r), r < n: T^g = occupied block; r >= n: active-virtual block)   (W7)
//   X0_g = tr T^g,  Ex0_g = tr(T^g T^g)
//   Bfull^g[r'][i] = Lam_v^g[r'][i] - sum_l Theta_v[r'][l] T^g[l][i]
//   B^g[x=(r',h)]  = Bfull^g[r'][pos(h)]             -> Bp (complex rows; the V GEMM expands them to the real (br,-bi | bi,br) form itself)
//   FK[x]         += sum_l Bfull^g[r'][l] T^g[l][pos(h)]      (exchange-like part of F, W9)
//   slice g = n_chol holds h1: Hrot[x] = B^{h1}[x], E1_0 += tr T^{h1}                              (W8)
// CTA = (chunk of GC slices, walker, spin).
// ------------------------------------------------------------------------------------------------
template <int GC>
__global__ void __launch_bounds__(256)
k_energy_dense(int n_chol, int64_t nw, SpinDev sa, SpinDev sb, const cplx* __restrict__ theta_a,
               const cplx* __restrict__ theta_b, const cplx* __restrict__ Lam_a, const cplx* __restrict__ Lam_b,
               cplx* Bp_a, cplx* Bp_b, cplx* X0 /*[2][nw][n_chol]*/, cplx* F_a, cplx* F_b,
               cplx* Hrot_a, cplx* Hrot_b, cplx* Eacc, int N)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int s = blockIdx.z;
    const int64_t w = blockIdx.y;
    const int g0 = blockIdx.x * GC;
    const SpinDev sp = s ? sb : sa;
    const int n = sp.n, no = sp.n_o, nv = sp.n_v, nr = sp.n_r, P = sp.P;
    if (n == 0) return;
    const cplx* theta = (s ? theta_b : theta_a) + w * (int64_t)N * n;
    const cplx* Lam = s ? Lam_b : Lam_a;
    cplx* Bp = (s ? Bp_b : Bp_a) + w * (int64_t)P * n_chol;
    cplx* F = (s ? F_b : F_a) + w * (int64_t)P;
    cplx* Hrot = (s ? Hrot_b : Hrot_a) + w * (int64_t)P;
    const int tid = threadIdx.x, nt = blockDim.x;

    cplx* T = reinterpret_cast<cplx*>(smem_raw);     // [n][n]
    cplx* Bf = T + n * n;                             // [nv][n]   Lam_v then Bfull (in place)
    cplx* Thv = Bf + nv * n;                          // [nv][n]   Theta rows of the active virtuals
    cplx* Fk = Thv + nv * n;                          // [P]       accumulates sum_g BT^g
    cplx* Bout = Fk + P;                              // [P][GC]
    int* pos = reinterpret_cast<int*>(Bout + (size_t)P * GC);   // [no]

    for (int e = tid; e < nv * n; e += nt) { int r = e / n, l = e - r * n; Thv[e] = theta[(int64_t)sp.act_v[r] * n + l]; }
    for (int x = tid; x < P; x += nt) Fk[x] = cmake(0.0, 0.0);
    for (int h = tid; h < no; h += nt) pos[h] = sp.pos_o[h];
    cplx ex_part = cmake(0.0, 0.0);
    __syncthreads();

    for (int gi = 0; gi < GC; gi++) {
        const int g = g0 + gi;
        if (g > n_chol) {                  // past the h1 slice: pad Bout
            for (int x = tid; x < P; x += nt) Bout[(size_t)x * GC + gi] = cmake(0.0, 0.0);
            continue;
        }
        const cplx* lam = Lam + ((int64_t)g * nr * nw + w) * n;      // row r at + r * nw * n
        for (int e = tid; e < nr * n; e += nt) {
            int r = e / n, i = e - r * n;
            cplx v = lam[(int64_t)r * nw * n + i];
            if (r < n) T[e] = v; else Bf[(r - n) * n + i] = v;
        }
        __syncthreads();
        // X0, Ex0 (the h1 slice contributes tr T to E1_0 instead)
        if (tid < 32) {
            cplx tr = cmake(0.0, 0.0);
            for (int l = tid; l < n; l += 32) tr = cadd(tr, T[l * n + l]);
            for (int o = 16; o > 0; o >>= 1) {
                tr.x += __shfl_down_sync(0xffffffffu, tr.x, o);
                tr.y += __shfl_down_sync(0xffffffffu, tr.y, o);
            }
            if (tid == 0) {
                if (g < n_chol) X0[((int64_t)s * nw + w) * n_chol + g] = tr;
                else red_add(&Eacc[w * 2 + 0], tr);
            }
        }
        if (g < n_chol)
            for (int e = tid; e < n * n; e += nt) { int l = e / n, i = e - l * n; ex_part = cfma(T[e], T[i * n + l], ex_part); }
        // Bfull = Lam_v - Theta_v T
        for (int e = tid; e < nv * n; e += nt) {
            int r = e / n, i = e - r * n;
            cplx acc = Bf[e];
            const cplx* tv = Thv + r * n;
            for (int l = 0; l < n; l++) acc = cfms(tv[l], T[l * n + i], acc);
            // the element is only read by its own thread before the barrier
            Bf[e] = acc;
        }
        __syncthreads();
        for (int x = tid; x < P; x += nt) {
            int r = x / no, h = x - r * no;
            const int ph = pos[h];
            cplx b = Bf[r * n + ph];
            Bout[(size_t)x * GC + gi] = b;
            if (g < n_chol) {
                cplx acc = cmake(0.0, 0.0);
                const cplx* bf = Bf + r * n;
                for (int l = 0; l < n; l++) acc = cfma(bf[l], T[l * n + ph], acc);
                Fk[x] = cadd(Fk[x], acc);
            } else {
                Hrot[x] = b;
            }
        }
        __syncthreads();
    }
    // flush: B rows (GC consecutive slices per x), exchange part of F, Ex0
    const int gcount = (g0 + GC <= n_chol) ? GC : (n_chol - g0 > 0 ? n_chol - g0 : 0);
    for (int e = tid; e < P * GC; e += nt) {
        int x = e / GC, gi = e - x * GC;
        if (gi >= gcount) continue;
        cplx b = Bout[e];
        const int g = g0 + gi;
        Bp[(int64_t)x * n_chol + g] = b;
    }
    for (int x = tid; x < P; x += nt) red_add(&F[x], cneg(Fk[x]));
    cplx ex = block_sum(ex_part);
    if (tid == 0) red_add(&Eacc[w * 2 + 1], cscale(-0.5, ex));
}

// ------------------------------------------------------------------------------------------------
// S7 on the FP64 tensor cores: the same quantities as k_energy_dense (which stays as the fallback for active windows
// wider than 16 x 16), with the two small complex products of every (walker, spin, slice) written as real DMMA
// m8n8k4 tiles.  One WARP owns one Cholesky slice g at a time; a CTA = (chunk of slices, walker, spin).
//   step 2   Bfull = Lam_v - Theta_v T        [Re; Im](2 n_v x n)  =  Lam_v + A'(2 n_v x 2n) B'(2n x n)
//            A'[r][2l+c]       = -(Theta_r, -Theta_i)[c]   (Re rows)     B'[2l+c][i] = (T_r, T_i)[c]
//            A'[half + r][2l+c] = -(Theta_i,  Theta_r)[c]   (Im rows)
//   step 4   FK += Bfull T[:, pos]              A''[r][2l+c] = (B_r, -B_i)[c] / (B_i, B_r)[c] read straight from the
//                                               complex Bfull tile with a per-lane component swap and sign
// Shared-memory strides are chosen so that every fragment load is a minimal 2-wavefront access.
// ------------------------------------------------------------------------------------------------
struct DenseMmaLayout {
    int half;      // n_v rounded up to 8: Im rows of the stacked outputs start here
    int Kp;        // 2n rounded up to 4
    int lda;       // row stride of A'     (doubles), = 4 mod 8
    int ldt;       // row stride of T      (doubles), = 8 mod 16
    int ldb;       // row stride of Lam_v  (doubles), = 4 mod 8
    int trows;     // rows of the T buffer (n, +1 zero row if n is odd)
    int warp_doubles;   // per-warp buffer: T then Lam_v/Bfull (+ slack for padded-tile over-reads)
    __host__ __device__ static int up(int v, int m, int r) { while (v % m != r) v++; return v; }
    __host__ __device__ DenseMmaLayout(int n, int nv) {
        half = (nv + 7) / 8 * 8;
        Kp = (2 * n + 3) / 4 * 4;
        lda = up(Kp, 8, 4);
        ldt = up(2 * n, 16, 8);
        ldb = up(Kp, 8, 4);
        trows = Kp / 2;
        warp_doubles = trows * ldt + half * ldb + 64;
        if (warp_doubles < 2 * half * 16) warp_doubles = 2 * half * 16;     // the FK partials alias this buffer
    }
};

// MTC / NTC > 0 fix the row-tile and column-tile counts at compile time (the common shapes: every guard and tile loop of the
// DMMA steps folds away); 0 keeps them as run-time values.
template <int NWARP, int MTC, int NTC>
__global__ void __launch_bounds__(NWARP * 32, NWARP == 8 ? 2 : 3)
k_energy_dense_mma(int n_chol, int64_t nw, int gchunk, SpinDev sa, SpinDev sb, const cplx* __restrict__ theta_a,
                   const cplx* __restrict__ theta_b, const cplx* __restrict__ Lam_a, const cplx* __restrict__ Lam_b,
                   cplx* Bp_a, cplx* Bp_b, cplx* X0 /*[2][nw][n_chol]*/, cplx* F_a, cplx* F_b,
                   cplx* Hrot_a, cplx* Hrot_b, cplx* Eacc, int N)
{
    extern __shared__ __align__(16) double smd[];
    const int s = blockIdx.z;
    const int64_t w = blockIdx.y;
    const SpinDev sp = s ? sb : sa;
    const int n = sp.n, no = sp.n_o, nv = sp.n_v, nr = sp.n_r, P = sp.P;
    if (n == 0) return;
    const DenseMmaLayout L(n, nv);
    const cplx* theta = (s ? theta_b : theta_a) + w * (int64_t)N * n;
    const cplx* Lam = s ? Lam_b : Lam_a;
    cplx* Bp = (s ? Bp_b : Bp_a) + w * (int64_t)P * n_chol;
    cplx* F = (s ? F_b : F_a) + w * (int64_t)P;
    cplx* Hrot = (s ? Hrot_b : Hrot_a) + w * (int64_t)P;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int gq = lane >> 2, tq = lane & 3;

    double* Ap = smd;                                         // [2 half][lda]
    double* wbuf = Ap + 2 * L.half * L.lda + wid * L.warp_doubles;
    double* Tb = wbuf;                                        // [trows][ldt]   (i, c) interleaved
    double* Lb = wbuf + L.trows * L.ldt;                      // [half][ldb]    Lam_v, then Bfull in place
    int* pos = reinterpret_cast<int*>(Ap + 2 * L.half * L.lda + NWARP * L.warp_doubles);   // [16]

    // zero everything once (padding must stay finite: padded K columns multiply zero rows)
    {
        const int tot = 2 * L.half * L.lda + NWARP * L.warp_doubles;
        for (int e = tid; e < tot; e += NWARP * 32) smd[e] = 0.0;
        if (tid < 16) pos[tid] = tid < no ? sp.pos_o[tid] : 0;
    }
    __syncthreads();
    for (int e = tid; e < nv * n; e += NWARP * 32) {
        const int r = e / n, l = e - r * n;
        const cplx t = theta[(int64_t)sp.act_v[r] * n + l];
        Ap[r * L.lda + 2 * l] = -t.x;            Ap[r * L.lda + 2 * l + 1] = t.y;
        Ap[(L.half + r) * L.lda + 2 * l] = -t.y; Ap[(L.half + r) * L.lda + 2 * l + 1] = -t.x;
    }
    __syncthreads();

    const int MT = MTC > 0 ? MTC : 2 * L.half / 8;            // <= 4
    const int NT = NTC > 0 ? NTC : (n + 7) / 8;
    const int KS = L.Kp / 4;
    // per-lane constants of the step-4 fragments
    const int posh[2] = {pos[gq], pos[8 + gq]};
    const int kc = tq & 1, kl = tq >> 1;      // k = 4 kk + tq  ->  l = 2 kk + kl, component kc
    double fk[4][2][2];
#pragma unroll
    for (int a = 0; a < 4; a++)
#pragma unroll
        for (int b = 0; b < 2; b++) { fk[a][b][0] = 0.0; fk[a][b][1] = 0.0; }
    cplx ex_part = cmake(0.0, 0.0);

    // step-4 A'' fragments: row m = 8 mt + gq of the stacked (Re; Im) operand reads component (kc ^ im) of Bfull[r][2kk+kl],
    // negated for Re rows with kc = 1
    int a4off[4];
    long long a4sgn[4];
#pragma unroll
    for (int mt = 0; mt < 4; mt++) {
        const int m = 8 * mt + gq, im = m >= L.half, r = m - im * L.half;
        a4off[mt] = r * L.ldb + 2 * kl + (kc ^ im);
        a4sgn[mt] = (!im && kc) ? (long long)0x8000000000000000ull : 0ll;
    }
    // output phase: element offset of pair index x = tid / NWARP + 32 t inside a warp's Bfull tile (P <= 256: 8 values)
    int ooff[8];
#pragma unroll
    for (int t = 0; t < 8; t++) {
        const int x = tid / NWARP + 32 * t;
        const int r = x / no, h = x - r * no;
        ooff[t] = (x < P) ? r * L.ldb + 2 * pos[h] : 0;
    }
    const int g_begin = blockIdx.x * gchunk;
    const int g_end = min(g_begin + gchunk, n_chol + 1);
    for (int g0 = g_begin; g0 < g_end; g0 += NWARP) {
        const int g = g0 + wid;
        const bool live = g < g_end;
        if (live) {
            // stage T^g (rows l < n) and Lam_v^g (rows n + r) of this walker: n complex = 2n doubles per row
            const cplx* lam = Lam + ((int64_t)g * nr * nw + w) * n;
            for (int i = lane; i < n; i += 32) {               // (no integer division in the per-slice loops)
                for (int r = 0; r < n; r++) cp_async16(Tb + r * L.ldt + 2 * i, lam + (int64_t)r * nw * n + i, 16);
                for (int r = n; r < nr; r++) cp_async16(Lb + (r - n) * L.ldb + 2 * i, lam + (int64_t)r * nw * n + i, 16);
            }
            cp_async_commit();
            cp_async_wait<0>();
        }
        __syncwarp();
        if (live) {
            // X0 = tr T, Ex0 += sum T[l][i] T[i][l]
            cplx tr = cmake(0.0, 0.0);
            for (int l = lane; l < n; l += 32) tr = cadd(tr, cmake(Tb[l * L.ldt + 2 * l], Tb[l * L.ldt + 2 * l + 1]));
            if (g < n_chol)
                // sum_{l,i} T[l][i] T[i][l], lane = i; the column read T[i][.] is skewed by i so that the lanes of a
                // warp do not all hit the two banks that the row stride (= 8 mod 16 doubles) maps a column to
                for (int i = lane; i < n; i += 32) {
                    int l = i;
                    for (int t = 0; t < n; t++) {
                        ex_part = cfma(cmake(Tb[l * L.ldt + 2 * i], Tb[l * L.ldt + 2 * i + 1]),
                                       cmake(Tb[i * L.ldt + 2 * l], Tb[i * L.ldt + 2 * l + 1]), ex_part);
                        l = (l + 1 == n) ? 0 : l + 1;
                    }
                }
            for (int o = 16; o > 0; o >>= 1) {
                tr.x += __shfl_down_sync(0xffffffffu, tr.x, o);
                tr.y += __shfl_down_sync(0xffffffffu, tr.y, o);
            }
            if (lane == 0) {
                if (g < n_chol) X0[((int64_t)s * nw + w) * n_chol + g] = tr;
                else red_add(&Eacc[w * 2 + 0], tr);
            }
            // step 2: Bfull = Lam_v + A' B', n-tiles in chunks of 3
            for (int nt0 = 0; nt0 < NT; nt0 += 3) {
                double acc[4][3][2];
#pragma unroll
                for (int mt = 0; mt < 4; mt++) {
                    const int m = 8 * mt + gq, im = m >= L.half, r = m - im * L.half;
#pragma unroll
                    for (int j = 0; j < 3; j++) {
                        const int i = 8 * (nt0 + j) + 2 * tq;
                        const bool ok = mt < MT && r < nv;
                        acc[mt][j][0] = (ok && i < n) ? Lb[r * L.ldb + 2 * i + im] : 0.0;
                        acc[mt][j][1] = (ok && i + 1 < n) ? Lb[r * L.ldb + 2 * i + 2 + im] : 0.0;
                    }
                }
                for (int kk = 0; kk < KS; kk++) {
                    double a[4], b[3];
#pragma unroll
                    for (int mt = 0; mt < 4; mt++) a[mt] = mt < MT ? Ap[(8 * mt + gq) * L.lda + 4 * kk + tq] : 0.0;
#pragma unroll
                    for (int j = 0; j < 3; j++)
                        b[j] = (nt0 + j < NT) ? Tb[(2 * kk + kl) * L.ldt + 2 * (8 * (nt0 + j) + gq) + kc] : 0.0;
#pragma unroll
                    for (int mt = 0; mt < 4; mt++)
#pragma unroll
                        for (int j = 0; j < 3; j++) dmma884(acc[mt][j][0], acc[mt][j][1], a[mt], b[j]);
                }
#pragma unroll
                for (int mt = 0; mt < 4; mt++) {
                    const int m = 8 * mt + gq, im = m >= L.half, r = m - im * L.half;
#pragma unroll
                    for (int j = 0; j < 3; j++) {
                        const int i = 8 * (nt0 + j) + 2 * tq;
                        const bool ok = mt < MT && r < nv;
                        if (ok && i < n) Lb[r * L.ldb + 2 * i + im] = acc[mt][j][0];
                        if (ok && i + 1 < n) Lb[r * L.ldb + 2 * i + 2 + im] = acc[mt][j][1];
                    }
                }
            }
        }
        __syncwarp();
        if (live && g < n_chol) {
            // step 4: FK += A''(Bfull) B''(T[:, pos])
            for (int kk = 0; kk < KS; kk++) {
                double a[4], b[2];
#pragma unroll
                for (int mt = 0; mt < 4; mt++) {
                    // offsets and sign masks are per-lane constants (a4off / a4sgn); the sign flip is an integer XOR so
                    // that no DADD competes with the DMMAs for the FP64 pipe
                    const double v = mt < MT ? Lb[a4off[mt] + 4 * kk] : 0.0;
                    a[mt] = __longlong_as_double(__double_as_longlong(v) ^ a4sgn[mt]);
                }
#pragma unroll
                for (int j = 0; j < 2; j++) b[j] = Tb[(2 * kk + kl) * L.ldt + 2 * posh[j] + kc];
#pragma unroll
                for (int mt = 0; mt < 4; mt++)
#pragma unroll
                    for (int j = 0; j < 2; j++) dmma884(fk[mt][j][0], fk[mt][j][1], a[mt], b[j]);
            }
        }
        __syncthreads();
        // cooperative output of the round's slices: thread (x, gi) -> NWARP consecutive slices of one pair index
        {
            const int gcount = min(NWARP, g_end - g0);
            const int gi = tid % NWARP;                        // thread (x, gi): x = tid / NWARP + 32 t
#pragma unroll
            for (int t = 0; t < 8; t++) {
                const int x = tid / NWARP + 32 * t;
                if (x >= P || gi >= gcount) continue;
                const int g = g0 + gi;
                const double* lb = Ap + 2 * L.half * L.lda + gi * L.warp_doubles + L.trows * L.ldt;
                const cplx b = cmake(lb[ooff[t]], lb[ooff[t] + 1]);
                if (g < n_chol) {
                    Bp[(int64_t)x * n_chol + g] = b;
                } else {
                    Hrot[x] = b;
                }
            }
        }
        __syncthreads();
    }

    // FK: sum the warps' partial tiles, then F -= FK (exchange-like part of F, W9); Ex0
    double* red = Ap + 2 * L.half * L.lda;                   // aliases the warp buffers (all reads are done)
#pragma unroll
    for (int mt = 0; mt < 4; mt++)
#pragma unroll
        for (int j = 0; j < 2; j++) {
            if (mt >= MT) continue;
            double* dst = red + ((wid * 2 * L.half) + 8 * mt + gq) * 16 + 8 * j + 2 * tq;
            dst[0] = fk[mt][j][0]; dst[1] = fk[mt][j][1];
        }
    __syncthreads();
    for (int x = tid; x < P; x += NWARP * 32) {
        const int r = x / no, h = x - r * no;
        double re = 0.0, im = 0.0;
        for (int ww = 0; ww < NWARP; ww++) {
            re += red[((ww * 2 * L.half) + r) * 16 + h];
            im += red[((ww * 2 * L.half) + L.half + r) * 16 + h];
        }
        red_add(&F[x], cmake(-re, -im));
    }
    cplx ex = block_sum(ex_part);
    if (tid == 0) red_add(&Eacc[w * 2 + 1], cscale(-0.5, ex));
}

// ------------------------------------------------------------------------------------------------
// S7 fused: the half rotation Lam^g = L_sub^g Theta and everything k_energy_dense_mma derives from it in ONE kernel, so that
// Lam (1.8 GB at fe2s2) is never written to or read from HBM.  A warp owns slice g of walker w: it computes the n_r x n
// complex tile Lam^g by FP64 DMMA (MTG x NTG tiles of 8x8, accumulators in registers; its rows of L_sub stream through a
// per-warp two-stage cp.async buffer, the walker's Theta^T operand sits in shared memory for the whole CTA), drops the tile
// into its T / Lam_v buffers and carries on with the dense steps of k_energy_dense_mma (X0, Ex0, Bfull, FK) on the same data.
// When the reference occupies the first n orbitals (n even), Theta[occ rows] is the identity, so the contraction runs over the
// N - n virtual orbitals only and L_sub[g][r][occ_i] is added as a constant (20 % fewer flops at fe2s2).
// Shapes: MTG = ceil(n_r / 8) <= 5, NTG = ceil(2 n / 8) <= 6 as template parameters (a predicated-off DMMA costs as much as
// an executed one, so the tile counts must be compile-time); other shapes take the two-kernel path.
// ------------------------------------------------------------------------------------------------
#define FUSE_NWARP 4
#define FUSE_BK 16
#define FUSE_LDA 20
__host__ __device__ inline int fused_ldbs(int Kv) { return (Kv + 15) / 16 * 16 + 4; }
template <int NWARP, int MTC, int NTC, int MTG, int NTG, int KSC>
__global__ void __launch_bounds__(NWARP * 32, NWARP == 8 ? 1 : 2)
k_energy_fused(int n_chol, int64_t nw, int gchunk, int ldN, int koff, int Kv, SpinDev sa, SpinDev sb,
               const cplx* __restrict__ theta_a, const cplx* __restrict__ theta_b, const double* __restrict__ thT_a,
               const double* __restrict__ thT_b, cplx* Bp_a, cplx* Bp_b, cplx* X0 /*[2][nw][n_chol]*/, cplx* F_a, cplx* F_b,
               cplx* Hrot_a, cplx* Hrot_b, cplx* Eacc, int N)
{
    extern __shared__ __align__(16) double smd[];
    const int s = blockIdx.z;
    const int64_t w = blockIdx.y;
    const SpinDev sp = s ? sb : sa;
    const int n = sp.n, no = sp.n_o, nv = sp.n_v, nr = sp.n_r, P = sp.P;
    if (n == 0) return;
    const DenseMmaLayout L(n, nv);
    const cplx* theta = (s ? theta_b : theta_a) + w * (int64_t)N * n;
    const double* thT = (s ? thT_b : thT_a) + w * (int64_t)n * 2 * ldN;     // rows (i, c), K = q contiguous
    const double* Lsub = sp.Lsub;
    cplx* Bp = (s ? Bp_b : Bp_a) + w * (int64_t)P * n_chol;
    cplx* F = (s ? F_b : F_a) + w * (int64_t)P;
    cplx* Hrot = (s ? Hrot_b : Hrot_a) + w * (int64_t)P;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int gq = lane >> 2, tq = lane & 3;

    const int wdoubles = max(L.warp_doubles, 2 * 8 * MTG * FUSE_LDA);     // per-warp buffer: T + Lam_v, aliased by the A stages
    const int Kvp = (Kv + 3) & ~3;                            // k4-steps; loads beyond Kv are zero-filled
    const int ldbs = fused_ldbs(Kv);                          // row stride of the Theta^T operand (= 4 mod 16: conflict-free)
    double* Ap = smd;                                         // [2 half][lda]
    double* wbase = Ap + 2 * L.half * L.lda;
    double* wbuf = wbase + wid * wdoubles;
    double* Tb = wbuf;                                        // [trows][ldt]   (i, c) interleaved
    double* Lb = wbuf + L.trows * L.ldt;                      // [half][ldb]    Lam_v, then Bfull in place
    double* Bs = wbase + NWARP * wdoubles;                    // [8 NTG][ldbs]  Theta^T columns (i, c) x virtual orbitals
    int* pos = reinterpret_cast<int*>(Bs + 8 * NTG * ldbs);   // [16]

    {
        const int tot = 2 * L.half * L.lda + NWARP * wdoubles + 8 * NTG * ldbs;
        for (int e = tid; e < tot; e += NWARP * 32) smd[e] = 0.0;
        if (tid < 16) pos[tid] = tid < no ? sp.pos_o[tid] : 0;
    }
    __syncthreads();
    for (int e = tid; e < nv * n; e += NWARP * 32) {
        const int r = e / n, l = e - r * n;
        const cplx t = theta[(int64_t)sp.act_v[r] * n + l];
        Ap[r * L.lda + 2 * l] = -t.x;            Ap[r * L.lda + 2 * l + 1] = t.y;
        Ap[(L.half + r) * L.lda + 2 * l] = -t.y; Ap[(L.half + r) * L.lda + 2 * l + 1] = -t.x;
    }
    for (int e = tid; e < 2 * n * Kv; e += NWARP * 32) {
        const int col = e / Kv, k = e - col * Kv;
        Bs[col * ldbs + k] = (koff + k < ldN) ? thT[(int64_t)col * ldN + koff + k] : 0.0;
    }
    __syncthreads();

    const int MT = MTC > 0 ? MTC : 2 * L.half / 8;            // <= 4
    const int NT = NTC > 0 ? NTC : (n + 7) / 8;
    constexpr int KS = KSC;                                   // = Kp / 4 (checked by the launcher)
    const int posh[2] = {pos[gq], pos[8 + gq]};
    const int kc = tq & 1, kl = tq >> 1;
    double fk[4][2][2];
#pragma unroll
    for (int a = 0; a < 4; a++)
#pragma unroll
        for (int b = 0; b < 2; b++) { fk[a][b][0] = 0.0; fk[a][b][1] = 0.0; }
    cplx ex_part = cmake(0.0, 0.0);
    int a4off[4];
    long long a4sgn[4];
#pragma unroll
    for (int mt = 0; mt < 4; mt++) {
        const int m = 8 * mt + gq, im = m >= L.half, r = m - im * L.half;
        a4off[mt] = r * L.ldb + 2 * kl + (kc ^ im);
        a4sgn[mt] = (!im && kc) ? (long long)0x8000000000000000ull : 0ll;
    }
    int ooff[8];
#pragma unroll
    for (int t = 0; t < 8; t++) {
        const int x = tid / NWARP + 32 * t;
        const int r = x / no, h = x - r * no;
        ooff[t] = (x < P) ? r * L.ldb + 2 * pos[h] : 0;
    }
    const int g_begin = blockIdx.x * gchunk;
    const int g_end = min(g_begin + gchunk, n_chol + 1);
    const int nchunk = (Kvp + FUSE_BK - 1) / FUSE_BK;
    for (int g0 = g_begin; g0 < g_end; g0 += NWARP) {
        const int g = g0 + wid;
        const bool live = g < g_end;
        if (live) {
            // ---- Lam^g = L_sub^g[:, virtual columns] Theta_V (+ L_sub^g[:, occ columns]) by DMMA, accumulators in registers ----
            const double* Arow = Lsub + ((int64_t)g * nr) * ldN + koff;
            double* As = wbuf;                                 // [2][8 MTG][FUSE_LDA]  (aliases Tb / Lb: they are dead here)
            // lane -> (row lane / 8 + 4 t, 16-byte column lane % 8): plain pointer increments, no per-element index arithmetic
            const double* asrc = Arow + (int64_t)(lane >> 3) * ldN + (lane & 7) * 2;
            double* adst = As + (lane >> 3) * FUSE_LDA + (lane & 7) * 2;
            const int arows = (nr - (lane >> 3) + 3) >> 2;      // rows of this lane: lane / 8, lane / 8 + 4, ...
            auto load_chunk = [&](int st, int ck) {
                const int k0 = ck * FUSE_BK;
                const bool ok = k0 + (lane & 7) * 2 < Kv;
                const double* sp_ = asrc + k0;
                double* dp = adst + st * 8 * MTG * FUSE_LDA;
                for (int t = 0; t < arows; t++) {
                    cp_async16(dp, ok ? sp_ : Arow, ok ? 16 : 0);
                    sp_ += 4 * (int64_t)ldN; dp += 4 * FUSE_LDA;
                }
            };
            load_chunk(0, 0);
            cp_async_commit();
            // accumulators start from the occupied columns of L_sub (Theta[occ rows] = 1): thread holds (row 8i + gq, column 4j + tq);
            // these loads are in flight while the first chunk arrives
            double acc[MTG][NTG][2];
#pragma unroll
            for (int i = 0; i < MTG; i++)
#pragma unroll
                for (int j = 0; j < NTG; j++) {
                    const int r = 8 * i + gq, ic = 4 * j + tq;
                    acc[i][j][0] = (koff && r < nr && ic < n) ? __ldg(Lsub + ((int64_t)g * nr + r) * ldN + ic) : 0.0;
                    acc[i][j][1] = 0.0;
                }
            for (int ck = 0; ck < nchunk; ck++) {
                if (ck + 1 < nchunk) load_chunk((ck + 1) & 1, ck + 1);
                cp_async_commit();
                cp_async_wait<1>();
                __syncwarp();
                const double* as = As + (ck & 1) * 8 * MTG * FUSE_LDA + gq * FUSE_LDA + tq;
                const double* bs = Bs + gq * ldbs + ck * FUSE_BK + tq;
                auto kstep = [&](int kk) {
                    double a[MTG], b[NTG];
#pragma unroll
                    for (int i = 0; i < MTG; i++) a[i] = as[i * 8 * FUSE_LDA + kk * 4];
#pragma unroll
                    for (int j = 0; j < NTG; j++) b[j] = bs[j * 8 * ldbs + kk * 4];
#pragma unroll
                    for (int i = 0; i < MTG; i++)
#pragma unroll
                        for (int j = 0; j < NTG; j++) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
                };
                const int ksteps = min(FUSE_BK, Kvp - ck * FUSE_BK) / 4;
                if (ksteps == FUSE_BK / 4) {       // full chunk: straight-line code, fragment loads of step k+1 overlap the DMMAs of step k
#pragma unroll
                    for (int kk = 0; kk < FUSE_BK / 4; kk++) kstep(kk);
                } else {
#pragma unroll 1
                    for (int kk = 0; kk < ksteps; kk++) kstep(kk);
                }
                __syncwarp();          // the stage is overwritten by the load issued in the next iteration
            }
            cp_async_wait<0>();
            __syncwarp();
            // accumulators -> T (rows < n) and Lam_v (rows n .. n_r)
#pragma unroll
            for (int i = 0; i < MTG; i++) {
                const int r = 8 * i + gq;
#pragma unroll
                for (int j = 0; j < NTG; j++) {
                    const int ic = 4 * j + tq;
                    if (r < nr && ic < n) {
                        double* dst = (r < n) ? Tb + r * L.ldt + 2 * ic : Lb + (r - n) * L.ldb + 2 * ic;
                        *reinterpret_cast<double2*>(dst) = make_double2(acc[i][j][0], acc[i][j][1]);
                    }
                }
            }
        }
        __syncwarp();
        if (live) {
            // X0 = tr T, Ex0 += sum T[l][i] T[i][l]
            cplx tr = cmake(0.0, 0.0);
            for (int l = lane; l < n; l += 32) tr = cadd(tr, cmake(Tb[l * L.ldt + 2 * l], Tb[l * L.ldt + 2 * l + 1]));
            if (g < n_chol)
                for (int i = lane; i < n; i += 32) {
                    int l = i;
                    cplx e1 = cmake(0.0, 0.0);                 // second chain: the FMA latency is not on the critical path
                    for (int t = 0; t + 1 < n; t += 2) {
                        const int l2 = (l + 1 == n) ? 0 : l + 1;
                        ex_part = cfma(*reinterpret_cast<const cplx*>(Tb + l * L.ldt + 2 * i),
                                       *reinterpret_cast<const cplx*>(Tb + i * L.ldt + 2 * l), ex_part);
                        e1 = cfma(*reinterpret_cast<const cplx*>(Tb + l2 * L.ldt + 2 * i),
                                  *reinterpret_cast<const cplx*>(Tb + i * L.ldt + 2 * l2), e1);
                        l = (l2 + 1 == n) ? 0 : l2 + 1;
                    }
                    if (n & 1)
                        e1 = cfma(*reinterpret_cast<const cplx*>(Tb + l * L.ldt + 2 * i),
                                  *reinterpret_cast<const cplx*>(Tb + i * L.ldt + 2 * l), e1);
                    ex_part = cadd(ex_part, e1);
                }
            for (int o = 16; o > 0; o >>= 1) {
                tr.x += __shfl_down_sync(0xffffffffu, tr.x, o);
                tr.y += __shfl_down_sync(0xffffffffu, tr.y, o);
            }
            if (lane == 0) {
                if (g < n_chol) X0[((int64_t)s * nw + w) * n_chol + g] = tr;
                else red_add(&Eacc[w * 2 + 0], tr);
            }
            // step 2: Bfull = Lam_v + A' B', n-tiles in chunks of 3
            for (int nt0 = 0; nt0 < NT; nt0 += 3) {
                double acc2[4][3][2];
#pragma unroll
                for (int mt = 0; mt < 4; mt++) {
                    const int m = 8 * mt + gq, im = m >= L.half, r = m - im * L.half;
#pragma unroll
                    for (int j = 0; j < 3; j++) {
                        const int i = 8 * (nt0 + j) + 2 * tq;
                        const bool ok = mt < MT && r < nv;
                        acc2[mt][j][0] = (ok && i < n) ? Lb[r * L.ldb + 2 * i + im] : 0.0;
                        acc2[mt][j][1] = (ok && i + 1 < n) ? Lb[r * L.ldb + 2 * i + 2 + im] : 0.0;
                    }
                }
#pragma unroll
                for (int kk = 0; kk < KS; kk++) {
                    double a[4], b[3];
#pragma unroll
                    for (int mt = 0; mt < 4; mt++) a[mt] = mt < MT ? Ap[(8 * mt + gq) * L.lda + 4 * kk + tq] : 0.0;
#pragma unroll
                    for (int j = 0; j < 3; j++)
                        b[j] = (nt0 + j < NT) ? Tb[(2 * kk + kl) * L.ldt + 2 * (8 * (nt0 + j) + gq) + kc] : 0.0;
#pragma unroll
                    for (int mt = 0; mt < 4; mt++)
#pragma unroll
                        for (int j = 0; j < 3; j++)
                            if (mt < MT && nt0 + j < NT) dmma884(acc2[mt][j][0], acc2[mt][j][1], a[mt], b[j]);
                }
#pragma unroll
                for (int mt = 0; mt < 4; mt++) {
                    const int m = 8 * mt + gq, im = m >= L.half, r = m - im * L.half;
#pragma unroll
                    for (int j = 0; j < 3; j++) {
                        const int i = 8 * (nt0 + j) + 2 * tq;
                        const bool ok = mt < MT && r < nv;
                        if (ok && i < n) Lb[r * L.ldb + 2 * i + im] = acc2[mt][j][0];
                        if (ok && i + 1 < n) Lb[r * L.ldb + 2 * i + 2 + im] = acc2[mt][j][1];
                    }
                }
            }
        }
        __syncwarp();
        if (live && g < n_chol) {
            // step 4: FK += A''(Bfull) B''(T[:, pos])
#pragma unroll
            for (int kk = 0; kk < KS; kk++) {
                double a[4], b[2];
#pragma unroll
                for (int mt = 0; mt < 4; mt++) {
                    const double v = mt < MT ? Lb[a4off[mt] + 4 * kk] : 0.0;
                    a[mt] = __longlong_as_double(__double_as_longlong(v) ^ a4sgn[mt]);
                }
#pragma unroll
                for (int j = 0; j < 2; j++) b[j] = Tb[(2 * kk + kl) * L.ldt + 2 * posh[j] + kc];
#pragma unroll
                for (int mt = 0; mt < 4; mt++)
#pragma unroll
                    for (int j = 0; j < 2; j++)
                        if (mt < MT) dmma884(fk[mt][j][0], fk[mt][j][1], a[mt], b[j]);
            }
        }
        __syncthreads();
        {   // cooperative output of the round's slices: thread (x, gi) -> NWARP consecutive slices of one pair index
            const int gcount = min(NWARP, g_end - g0);
            const int gi = tid % NWARP;
#pragma unroll
            for (int t = 0; t < 8; t++) {
                const int x = tid / NWARP + 32 * t;
                if (x >= P || gi >= gcount) continue;
                const int gg = g0 + gi;
                const double* lb = wbase + gi * wdoubles + L.trows * L.ldt;
                const cplx b = cmake(lb[ooff[t]], lb[ooff[t] + 1]);
                if (gg < n_chol) Bp[(int64_t)x * n_chol + gg] = b;
                else Hrot[x] = b;
            }
        }
        __syncthreads();
    }

    // FK: sum the warps' partial tiles, then F -= FK (exchange-like part of F, W9); Ex0
    double* red = wbase;                                       // aliases the warp buffers (all reads are done)
#pragma unroll
    for (int mt = 0; mt < 4; mt++)
#pragma unroll
        for (int j = 0; j < 2; j++) {
            if (mt >= MT) continue;
            double* dst = red + ((wid * 2 * L.half) + 8 * mt + gq) * 16 + 8 * j + 2 * tq;
            dst[0] = fk[mt][j][0]; dst[1] = fk[mt][j][1];
        }
    __syncthreads();
    for (int x = tid; x < P; x += NWARP * 32) {
        const int r = x / no, h = x - r * no;
        double re = 0.0, im = 0.0;
        for (int ww = 0; ww < NWARP; ww++) {
            re += red[((ww * 2 * L.half) + r) * 16 + h];
            im += red[((ww * 2 * L.half) + L.half + r) * 16 + h];
        }
        red_add(&F[x], cmake(-re, -im));
    }
    cplx ex = block_sum(ex_part);
    if (tid == 0) red_add(&Eacc[w * 2 + 1], cscale(-0.5, ex));
}

// F[x] += sum_g Xt_g B^g[x]  (Coulomb-like part of F, W9);   one warp per x
__global__ void __launch_bounds__(256)
k_fx(int n_chol, int64_t nw, int Pa, int Pb, const cplx* __restrict__ X0, const cplx* __restrict__ Bp_a,
     const cplx* __restrict__ Bp_b, cplx* F_a, cplx* F_b)
{
    const int s = blockIdx.z;
    const int64_t w = blockIdx.y;
    const int P = s ? Pb : Pa;
    const int x = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (x >= P) return;
    const int lane = threadIdx.x & 31;
    const cplx* b = (s ? Bp_b : Bp_a) + (w * (int64_t)P + x) * n_chol;
    const cplx* xa = X0 + w * (int64_t)n_chol;
    const cplx* xb = X0 + (nw + w) * (int64_t)n_chol;
    cplx acc = cmake(0.0, 0.0);
    for (int g = lane; g < n_chol; g += 32) acc = cfma(cadd(xa[g], xb[g]), b[g], acc);
    for (int o = 16; o > 0; o >>= 1) {
        acc.x += __shfl_down_sync(0xffffffffu, acc.x, o);
        acc.y += __shfl_down_sync(0xffffffffu, acc.y, o);
    }
    if (lane == 0) { cplx* F = (s ? F_b : F_a) + w * (int64_t)P + x; *F = cadd(*F, acc); }
}

template <int NWARP, int MTC, int NTC>
static cudaError_t launch_dense_mma_t(msd_ctx* c, int64_t nw, Workspace& ws, size_t smem, cudaStream_t st)
{
    cudaError_t e = func_config(c, (const void*)k_energy_dense_mma<NWARP, MTC, NTC>, NWARP * 32, smem, nullptr);
    if (e != cudaSuccess) return e;
    const int gchunk = 4 * NWARP;
    dim3 grid((c->n_chol + 1 + gchunk - 1) / gchunk, (unsigned)nw, 2);
    k_energy_dense_mma<NWARP, MTC, NTC><<<grid, NWARP * 32, smem, st>>>(
        c->n_chol, nw, gchunk, c->dev(0), c->dev(1), ws.theta[0], ws.theta[1], ws.Lam[0], ws.Lam[1], ws.Bp[0], ws.Bp[1],
        ws.X0, ws.F[0], ws.F[1], ws.Hrot[0], ws.Hrot[1], ws.Eacc, c->N);
    return cudaGetLastError();
}

template <int NWARP>
static cudaError_t launch_dense_mma(msd_ctx* c, int64_t nw, Workspace& ws, size_t smem, cudaStream_t st)
{
    // compile-time tile counts when both spins (those with electrons) have the same ones
    int mt = -1, nt = -1;
    for (int s = 0; s < 2; s++) {
        const auto& sp = c->sp[s];
        if (sp.n == 0) continue;
        const int m = 2 * ((sp.n_v + 7) / 8 * 8) / 8, t = (sp.n + 7) / 8;
        if (mt == -1) { mt = m; nt = t; }
        else if (mt != m || nt != t) { mt = 0; nt = 0; }
    }
    if (mt == 4 && nt == 3) return launch_dense_mma_t<NWARP, 4, 3>(c, nw, ws, smem, st);
    if (mt == 4 && nt == 2) return launch_dense_mma_t<NWARP, 4, 2>(c, nw, ws, smem, st);
    if (mt == 4 && nt == 1) return launch_dense_mma_t<NWARP, 4, 1>(c, nw, ws, smem, st);
    if (mt == 2 && nt == 3) return launch_dense_mma_t<NWARP, 2, 3>(c, nw, ws, smem, st);
    if (mt == 2 && nt == 2) return launch_dense_mma_t<NWARP, 2, 2>(c, nw, ws, smem, st);
    if (mt == 2 && nt == 1) return launch_dense_mma_t<NWARP, 2, 1>(c, nw, ws, smem, st);
    return launch_dense_mma_t<NWARP, 0, 0>(c, nw, ws, smem, st);
}

// dynamic shared memory of k_energy_dense<GC> (the larger of the two spins)
size_t energy_dense_smem(const msd_ctx* c, int GC)
{
    size_t smem = 0;
    for (int s = 0; s < 2; s++) {
        const auto& sp = c->sp[s];
        size_t v = ((size_t)sp.n * sp.n + 2 * (size_t)sp.n_v * sp.n + (size_t)sp.P * (1 + GC) + 1) * sizeof(cplx) +
                   (size_t)(sp.n_o + 4) * sizeof(int);
        if (v > smem) smem = v;
    }
    return smem;
}

template <int NWARP, int MTC, int NTC, int MTG, int NTG, int KSC>
static cudaError_t launch_fused_t(msd_ctx* c, int64_t nw, Workspace& ws, int koff, int Kv, cudaStream_t st)
{
    for (int s = 0; s < 2; s++)
        if (c->sp[s].n > 0 && DenseMmaLayout(c->sp[s].n, c->sp[s].n_v).Kp / 4 != KSC) return cudaErrorNotSupported;
    const int ldN = c->N + (c->N & 1);
    size_t smem = 0;
    for (int s = 0; s < 2; s++) {
        const auto& sp = c->sp[s];
        if (sp.n == 0) continue;
        DenseMmaLayout L(sp.n, sp.n_v);
        const int wd = std::max(L.warp_doubles, 2 * 8 * MTG * FUSE_LDA);
        smem = std::max(smem, ((size_t)2 * L.half * L.lda + (size_t)NWARP * wd + (size_t)8 * NTG * fused_ldbs(Kv)) * sizeof(double) + 64);
    }
    if (smem > 227 * 1024) return cudaErrorNotSupported;
    cudaError_t e = func_config(c, (const void*)k_energy_fused<NWARP, MTC, NTC, MTG, NTG, KSC>, NWARP * 32, smem, nullptr);
    if (e != cudaSuccess) return e;
    const int gchunk = 64;
    dim3 grid((c->n_chol + 1 + gchunk - 1) / gchunk, (unsigned)nw, 2);
    k_energy_fused<NWARP, MTC, NTC, MTG, NTG, KSC><<<grid, NWARP * 32, smem, st>>>(
        c->n_chol, nw, gchunk, ldN, koff, Kv, c->dev(0), c->dev(1), ws.theta[0], ws.theta[1], ws.thetaT[0], ws.thetaT[1],
        ws.Bp[0], ws.Bp[1], ws.X0, ws.F[0], ws.F[1], ws.Hrot[0], ws.Hrot[1], ws.Eacc, c->N);
    return cudaGetLastError();
}

// true (and *koff, *Kv set) when the fused S7 kernel covers this trial: both spins with electrons share the tile counts and the
// shape is one of the instantiated ones
bool energy_fused_shape(const msd_ctx* c, int* mtc, int* ntc, int* mtg, int* ntg, int* koff, int* Kv)
{
    int a = -1, b = -1, m = -1, t = -1;
    bool contiguous = true;
    int nn = -1;
    for (int s = 0; s < 2; s++) {
        const auto& sp = c->sp[s];
        if (sp.n == 0) continue;
        if (sp.n_o > 16 || sp.n_v > 16 || sp.n > 24) return false;
        const int A = 2 * ((sp.n_v + 7) / 8 * 8) / 8, B = (sp.n + 7) / 8, M = (sp.n_r + 7) / 8, T = (2 * sp.n + 7) / 8;
        if (a == -1) { a = A; b = B; m = M; t = T; nn = sp.n; }
        else if (a != A || b != B || m != M || t != T) return false;
        if (sp.n != nn || (sp.n & 1)) contiguous = false;
        for (int l = 0; l < sp.n; l++) if (sp.occ_ref[l] != l) contiguous = false;
    }
    if (a == -1) return false;
    const bool have = (a == 4 && b == 3 && m == 5 && t == 5) || (a == 4 && b == 2 && m == 4 && t == 4) ||
                      (a == 4 && b == 2 && m == 4 && t == 3) || (a == 2 && b == 1 && m == 2 && t == 2);
    if (!have) return false;
    const int ksc = (a == 4 && b == 3) ? 10 : (a == 4 && t == 4) ? 8 : (a == 4) ? 6 : 4;
    for (int s = 0; s < 2; s++)
        if (c->sp[s].n > 0 && DenseMmaLayout(c->sp[s].n, c->sp[s].n_v).Kp / 4 != ksc) return false;
    const int ldN = c->N + (c->N & 1);
    *mtc = a; *ntc = b; *mtg = m; *ntg = t;
    *koff = contiguous ? nn : 0;
    *Kv = ldN - *koff;
    return true;
}

cudaError_t launch_energy_fused(msd_ctx* c, int64_t nw, Workspace& ws, cudaStream_t st)
{
    int a, b, m, t, koff, Kv;
    if (!energy_fused_shape(c, &a, &b, &m, &t, &koff, &Kv)) return cudaErrorNotSupported;
    cudaError_t e;
    if (a == 4 && b == 3) e = launch_fused_t<FUSE_NWARP, 4, 3, 5, 5, 10>(c, nw, ws, koff, Kv, st);          // n = 20 (fe2s2)
    else if (a == 4 && t == 4) e = launch_fused_t<FUSE_NWARP, 4, 2, 4, 4, 8>(c, nw, ws, koff, Kv, st);      // n = 16 (cu2o2)
    else if (a == 4) e = launch_fused_t<FUSE_NWARP, 4, 2, 4, 3, 6>(c, nw, ws, koff, Kv, st);                // n = 12 (sweep)
    else e = launch_fused_t<FUSE_NWARP, 2, 1, 2, 2, 4>(c, nw, ws, koff, Kv, st);                            // n = 8 (small)
    if (e == cudaSuccess) c->launches++;
    return e;
}

cudaError_t launch_energy_dense(msd_ctx* c, int64_t nw, Workspace& ws, cudaStream_t st)
{
    if (nw == 0) return cudaSuccess;
    // tensor-core kernel when both active windows fit its register tiles (n_o, n_v <= 16), scalar kernel otherwise
    bool mma_ok = true;
    size_t need[2] = {0, 0};     // shared memory with 8 / 4 warps
    for (int s = 0; s < 2; s++) {
        const auto& sp = c->sp[s];
        if (sp.n == 0) continue;
        if (sp.n_o > 16 || sp.n_v > 16) mma_ok = false;
        DenseMmaLayout L(sp.n, sp.n_v);
        for (int k = 0; k < 2; k++) {
            size_t v = ((size_t)2 * L.half * L.lda + (size_t)(k ? 4 : 8) * L.warp_doubles) * sizeof(double) + 64;
            if (v > need[k]) need[k] = v;
        }
    }
    cudaError_t e = cudaSuccess;
    if (mma_ok && need[0] <= 113 * 1024) e = launch_dense_mma<8>(c, nw, ws, need[0], st);
    else if (mma_ok && need[1] <= 227 * 1024) e = launch_dense_mma<4>(c, nw, ws, need[1], st);
    else {
        // slices per CTA: as many as fit next to the per-walker tiles (the paper's Cu2O2 window, 16 x 92, takes 4)
        int GC = 8;
        while (GC > 1 && energy_dense_smem(c, GC) > 227 * 1024) GC >>= 1;
        const size_t smem = energy_dense_smem(c, GC);
        if (smem > 227 * 1024) return cudaErrorInvalidConfiguration;     // excluded at setup (energy_ok)
        // X0 of a spin with no electrons must read as zero: ws.X0 lies in the region zeroed per call
        dim3 grid((c->n_chol + 1 + GC - 1) / GC, (unsigned)nw, 2);
        auto go = [&](auto kern) {
            cudaError_t e2 = func_config(c, (const void*)kern, 256, smem, nullptr);
            if (e2 != cudaSuccess) return e2;
            kern<<<grid, 256, smem, st>>>(c->n_chol, nw, c->dev(0), c->dev(1), ws.theta[0], ws.theta[1], ws.Lam[0], ws.Lam[1],
                                          ws.Bp[0], ws.Bp[1], ws.X0, ws.F[0], ws.F[1], ws.Hrot[0], ws.Hrot[1], ws.Eacc, c->N);
            return cudaGetLastError();
        };
        e = GC == 8 ? go(k_energy_dense<8>) : GC == 4 ? go(k_energy_dense<4>) : GC == 2 ? go(k_energy_dense<2>) : go(k_energy_dense<1>);
    }
    c->launches++;
    return e;
}

// Coulomb-like part of F (k_fx).  Independent of the V GEMMs that follow the dense kernel (both only read Bp), so the
// caller puts it on a side stream next to them: it is HBM-bound, they are tensor-bound.
cudaError_t launch_fx(msd_ctx* c, int64_t nw, Workspace& ws, cudaStream_t st)
{
    cplx* X0 = ws.X0;
    int Pmax = c->sp[0].P > c->sp[1].P ? c->sp[0].P : c->sp[1].P;
    if (nw == 0 || Pmax == 0) return cudaSuccess;
    dim3 g2((Pmax + 7) / 8, (unsigned)nw, 2);
    k_fx<<<g2, 256, 0, st>>>(c->n_chol, nw, c->sp[0].P, c->sp[1].P, X0, ws.Bp[0], ws.Bp[1], ws.F[0], ws.F[1]);
    c->launches++;
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// S9 / finishing kernels
// ------------------------------------------------------------------------------------------------
__global__ void k_finish_overlap(int64_t nw, const cplx* __restrict__ det0, const cplx* __restrict__ Wacc,
                                 int* wflags, cplx* ovlp, int* flags)
{
    int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= nw) return;
    cplx W = Wacc[w];
    int f = wflags[w];
    if (W.x == 0.0 && W.y == 0.0) f |= 2;
    cplx o = cmul(cmul(det0[w * 2], det0[w * 2 + 1]), W);
    if (f) o = cmake(nan_d(), nan_d());
    ovlp[w] = o;
    if (flags) flags[w] = f;
}

// NaN-fill outputs of flagged walkers (force bias / greens) and export flags
__global__ void k_finish_flags(int64_t nw, const cplx* __restrict__ Wacc, const int* __restrict__ wflags, cplx* out,
                               int64_t per_walker, int* flags)
{
    const int64_t w = blockIdx.x;
    cplx W = Wacc[w];
    int f = wflags[w];
    if (W.x == 0.0 && W.y == 0.0) f |= 2;
    if (threadIdx.x == 0 && flags) flags[w] = f;
    if (f && out)
        for (int64_t e = threadIdx.x; e < per_walker; e += blockDim.x) out[w * per_walker + e] = cmake(nan_d(), nan_d());
}

//   E1 = E1_0 + (1/W) E1nd,   E1nd = sum_s sum_x C^s[x] Hrot^s[x]  (accumulated per determinant in the dets kernels)   (W8)
//   E2 = 1/2 sum_g Xt_g^2 - 1/2 sum_g (Ex0^a_g + Ex0^b_g) + (1/W) E2nd,
//   E2nd = sum_s sum_x C^s[x] F^s[x] + second-order sums                                                          (W9)
__global__ void __launch_bounds__(256)
k_finish_energy(int n_chol, int64_t nw, double e0, const cplx* __restrict__ X0, const cplx* __restrict__ Eacc,
                const cplx* __restrict__ Wacc, const cplx* __restrict__ E1nd, const cplx* __restrict__ E2nd,
                const int* __restrict__ wflags, cplx* eout, int64_t estride, int* flags)
{
    const int64_t w = blockIdx.x;
    const int tid = threadIdx.x, nt = blockDim.x;
    cplx xx = cmake(0.0, 0.0);
    for (int g = tid; g < n_chol; g += nt) {
        cplx xt = cadd(X0[w * (int64_t)n_chol + g], X0[(nw + w) * (int64_t)n_chol + g]);
        xx = cfma(xt, xt, xx);
    }
    xx = block_sum(xx);
    if (tid == 0) {
        cplx W = Wacc[w];
        int f = wflags[w];
        if (W.x == 0.0 && W.y == 0.0) f |= 2;
        cplx E1, E2;
        if (f) { E1 = cmake(nan_d(), nan_d()); E2 = E1; }
        else {
            cplx Winv = cinv(W);
            E1 = cadd(Eacc[w * 2 + 0], cmul(E1nd[w], Winv));
            E2 = cadd(cadd(cscale(0.5, xx), Eacc[w * 2 + 1]), cmul(E2nd[w], Winv));
        }
        eout[w * estride + 0] = cmake(e0 + E1.x + E2.x, E1.y + E2.y);
        eout[w * estride + 1] = E1;
        eout[w * estride + 2] = E2;
        if (flags) flags[w] = f;
    }
}

cudaError_t launch_finish_overlap(msd_ctx* c, int64_t nw, Workspace& ws, cplx* ovlp, int* flags, cudaStream_t st)
{
    if (nw == 0) return cudaSuccess;
    k_finish_overlap<<<(unsigned)((nw + 127) / 128), 128, 0, st>>>(nw, ws.det0, ws.Wacc, ws.wflags, ovlp, flags);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_finish_flags(msd_ctx* c, int64_t nw, Workspace& ws, cplx* out, int64_t per_walker, int* flags,
                                cudaStream_t st)
{
    if (nw == 0) return cudaSuccess;
    k_finish_flags<<<(unsigned)nw, 128, 0, st>>>(nw, ws.Wacc, ws.wflags, out, per_walker, flags);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_finish_energy(msd_ctx* c, int64_t nw, Workspace& ws, cplx* e, int64_t estride, int* flags, cudaStream_t st)
{
    if (nw == 0) return cudaSuccess;
    cplx* X0 = ws.X0;
    k_finish_energy<<<(unsigned)nw, 256, 0, st>>>(c->n_chol, nw, c->e0, X0, ws.Eacc, ws.Wacc, ws.E1nd, ws.E2nd, ws.wflags,
                                                  e, estride, flags);
    c->launches++;
    return cudaGetLastError();
}

// Force bias from the energy path's intermediates:
//   fb[w][g] = sum_s [ X0^s[w][g] + (1/W) sum_x C^s[x][w] B^{s,g}[w][x] ]
// C planar [tile][x][2][WT], Bp [w][x][g] (g contiguous: coalesced over the threads), out row stride `ostride`.
#define FB_XT 1024
__global__ void __launch_bounds__(256)
k_fb_from_cb(int n_chol, int64_t nw, int Pa, int Pb, const double* __restrict__ C_a, const double* __restrict__ C_b,
             const cplx* __restrict__ Bp_a, const cplx* __restrict__ Bp_b, const cplx* __restrict__ X0,
             const cplx* __restrict__ Wacc, const int* __restrict__ wflags, cplx* out, int64_t ostride)
{
    __shared__ cplx Cs[FB_XT];                                  // one chunk of C^s at a time (any window size)
    const int64_t w = blockIdx.y;
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    const cplx W = Wacc[w];
    const bool bad = wflags[w] || (W.x == 0.0 && W.y == 0.0);
    cplx acc[2] = {cmake(0.0, 0.0), cmake(0.0, 0.0)};
    for (int s = 0; s < 2; s++) {
        const int P = s ? Pb : Pa;
        const double* C = (s ? C_b : C_a) + (w / MSD_WT) * (int64_t)P * 2 * MSD_WT + (w % MSD_WT);
        const cplx* B = (s ? Bp_b : Bp_a) + w * (int64_t)P * n_chol + g;
        for (int x0 = 0; x0 < P; x0 += FB_XT) {
            const int nx = min(FB_XT, P - x0);
            __syncthreads();
            for (int x = threadIdx.x; x < nx; x += blockDim.x) Cs[x] = load_planar(C, x0 + x);
            __syncthreads();
            if (g < n_chol && !bad) {
#pragma unroll 4
                for (int x = 0; x < nx; x++) acc[x & 1] = cfma(Cs[x], B[(int64_t)(x0 + x) * n_chol], acc[x & 1]);
            }
        }
    }
    if (g >= n_chol) return;
    if (bad) { out[w * ostride + g] = cmake(nan_d(), nan_d()); return; }
    const cplx t = cmul(cadd(acc[0], acc[1]), cinv(W));
    const cplx x0 = cadd(X0[w * (int64_t)n_chol + g], X0[(nw + w) * (int64_t)n_chol + g]);
    out[w * ostride + g] = cadd(x0, t);
}

cudaError_t launch_fb_from_cb(msd_ctx* c, int64_t nw, Workspace& ws, cplx* out, int64_t ostride, cudaStream_t st)
{
    if (nw == 0 || c->n_chol == 0) return cudaSuccess;
    const int Pa = c->sp[0].P, Pb = c->sp[1].P;
    dim3 grid((c->n_chol + 255) / 256, (unsigned)nw);
    k_fb_from_cb<<<grid, 256, 0, st>>>(c->n_chol, nw, Pa, Pb, ws.C[0], ws.C[1], ws.Bp[0],
                                                                          ws.Bp[1], ws.X0, ws.Wacc, ws.wflags, out, ostride);
    c->launches++;
    return cudaGetLastError();
}

// S1 "reference" (Wick step W1): per (walker, spin)
//   O0 = psi[occ_ref,:]  (Psi_T^+ phi of PAPER.md Eq. 13 for the reference determinant), pivoted LU,
//   det0 = det O0 (Eq. 13), Theta = psi O0^-1 (N x n), so that the reference Green's function of Eq. 14
//   is G0[occ_ref[l], q] = Theta[q, l]; active slice g[h, p] = Theta[p, pos(h)].
// One CTA per (walker, spin).  complex128 throughout.
#include "msd_internal.cuh"

__global__ void __launch_bounds__(128)
k_reference(int N, int ldN, SpinDev sa, SpinDev sb, int64_t nw, const cplx* __restrict__ phi_a,
            const cplx* __restrict__ phi_b, cplx* theta_a, cplx* theta_b, double* thetaT_a, double* thetaT_b,
            cplx* det0, cplx* g_a, cplx* g_b, int* wflags, int stage_psi)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int s = blockIdx.y;
    const int64_t w = blockIdx.x;
    const SpinDev sp = s ? sb : sa;
    const int n = sp.n;
    const cplx* psi = (s ? phi_b : phi_a) + w * (int64_t)N * n;
    cplx* theta = (s ? theta_b : theta_a) + w * (int64_t)N * n;
    double* thetaT = (s ? thetaT_b : thetaT_a);
    cplx* g = (s ? g_b : g_a) + (w / MSD_WT) * (int64_t)sp.P * MSD_WT + (w % MSD_WT);
    const int tid = threadIdx.x, nt = blockDim.x;

    if (w >= nw) {   // padding walker of the last tile: zero active slice so that its lanes compute on zeros
        for (int x = tid; x < sp.P; x += nt) g[(int64_t)x * MSD_WT] = cmake(0.0, 0.0);
        return;
    }
    cplx* lu = reinterpret_cast<cplx*>(smem_raw);          // [n][n]
    cplx* inv = lu + n * n;                                 // [n][n]
    int* piv = reinterpret_cast<int*>(inv + n * n);         // [n]
    int* vmap = piv + n;                                    // [N]  orbital -> active-virtual index or -1
    int* omap = vmap + N;                                   // [n]  position in occ_ref -> active-occupied index or -1
    // the walker block itself, rows padded to n + 1 complex (conflict-free column walks in the Theta product);
    // read once, coalesced -- the strided global reads psi[q*n + m] were the whole cost of this kernel
    const int lps = n + 1;
    cplx* psis = reinterpret_cast<cplx*>(smem_raw + ((((size_t)2 * n * n * sizeof(cplx) + (size_t)(2 * n + N) * sizeof(int)) + 15) / 16) * 16);
    __shared__ int s_p;
    __shared__ int s_sing;
    __shared__ double s_sign;

    for (int q = tid; q < N; q += nt) vmap[q] = -1;
    for (int l = tid; l < n; l += nt) { omap[l] = -1; piv[l] = l; }
    if (tid == 0) { s_sing = 0; s_sign = 1.0; }
    __syncthreads();
    for (int r = tid; r < sp.n_v; r += nt) vmap[sp.act_v[r]] = r;
    for (int h = tid; h < sp.n_o; h += nt) omap[sp.pos_o[h]] = h;
    if (stage_psi) {
        for (int e = tid; e < N * n; e += nt) {
            int q = e / n, i = e - q * n;
            psis[q * lps + i] = psi[e];
        }
        __syncthreads();
    }
    for (int e = tid; e < n * n; e += nt) {
        int l = e / n, i = e - l * n;
        lu[e] = stage_psi ? psis[sp.occ_ref[l] * lps + i] : psi[(int64_t)sp.occ_ref[l] * n + i];
    }
    __syncthreads();

    // --- LU with partial pivoting (rows), in shared memory ---
    for (int j = 0; j < n; j++) {
        if (tid < 32) {
            double best = -1.0; int bi = j;
            for (int i = j + tid; i < n; i += 32) { double v = cabs2(lu[i * n + j]); if (v > best) { best = v; bi = i; } }
            for (int o = 16; o > 0; o >>= 1) {
                double ob = __shfl_down_sync(0xffffffffu, best, o);
                int oi = __shfl_down_sync(0xffffffffu, bi, o);
                if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
            }
            if (tid == 0) { s_p = bi; if (!(best > 0.0)) s_sing = 1; }
        }
        __syncthreads();
        if (s_sing) break;
        const int p = s_p;
        if (p != j) {
            for (int c = tid; c < n; c += nt) { cplx t = lu[j * n + c]; lu[j * n + c] = lu[p * n + c]; lu[p * n + c] = t; }
            if (tid == 0) { int t = piv[j]; piv[j] = piv[p]; piv[p] = t; s_sign = -s_sign; }
        }
        __syncthreads();
        const cplx rinv = cinv(lu[j * n + j]);
        for (int i = j + 1 + tid; i < n; i += nt) lu[i * n + j] = cmul(lu[i * n + j], rinv);
        __syncthreads();
        const int m = n - j - 1;
        for (int e = tid; e < m * m; e += nt) {
            int i = j + 1 + e / m, c = j + 1 + e % m;
            lu[i * n + c] = cfms(lu[i * n + j], lu[j * n + c], lu[i * n + c]);
        }
        __syncthreads();
    }
    const bool sing = s_sing != 0;
    if (tid == 0) {
        cplx d = cmake(s_sign, 0.0);
        if (sing) d = cmake(0.0, 0.0);
        else for (int j = 0; j < n; j++) d = cmul(d, lu[j * n + j]);
        det0[w * 2 + s] = d;
        if (sing) atomicOr(&wflags[w], 1);
    }
    // --- inverse: column c of O0^-1 solves (P O0) x = P e_c : thread c does both substitutions ---
    if (!sing) {
        for (int c = tid; c < n; c += nt) {
            for (int i = 0; i < n; i++) {
                cplx sacc = cmake(piv[i] == c ? 1.0 : 0.0, 0.0);
                for (int k = 0; k < i; k++) sacc = cfms(lu[i * n + k], inv[k * n + c], sacc);
                inv[i * n + c] = sacc;
            }
            for (int i = n - 1; i >= 0; i--) {
                cplx sacc = inv[i * n + c];
                for (int k = i + 1; k < n; k++) sacc = cfms(lu[i * n + k], inv[k * n + c], sacc);
                inv[i * n + c] = cmul(sacc, cinv(lu[i * n + i]));
            }
        }
    }
    __syncthreads();
    // --- Theta = psi O0^-1 and its three layouts ---
    const double nanv = __longlong_as_double(0x7ff8000000000000LL);
    for (int e = tid; e < N * n; e += nt) {
        int l = e / N, q = e - l * N;            // consecutive threads -> consecutive q
        cplx acc = cmake(0.0, 0.0);
        if (sing) acc = cmake(nanv, nanv);
        else if (stage_psi) for (int m = 0; m < n; m++) acc = cfma(psis[q * lps + m], inv[m * n + l], acc);
        else for (int m = 0; m < n; m++) acc = cfma(psi[(int64_t)q * n + m], inv[m * n + l], acc);
        theta[(int64_t)q * n + l] = acc;
        if (thetaT) {
            double* tt = thetaT + ((w * n + l) * 2) * (int64_t)ldN;     // rows (w, l, re/im), K = q contiguous
            tt[q] = acc.x; tt[ldN + q] = acc.y;
            if (q == 0 && ldN > N) { tt[N] = 0.0; tt[ldN + N] = 0.0; }     // zero the even-stride pad
        }
        int r = vmap[q], h = omap[l];
        if (r >= 0 && h >= 0) g[(int64_t)(r * sp.n_o + h) * MSD_WT] = acc;
    }
}

cudaError_t launch_reference(msd_ctx* c, int N, int ldN, SpinDev sa, SpinDev sb, int64_t nw, const cplx* phi_a,
                             const cplx* phi_b, Workspace& ws, bool want_thetaT, cudaStream_t st)
{
    int nmax = sa.n > sb.n ? sa.n : sb.n;
    size_t smem = (size_t)2 * nmax * nmax * sizeof(cplx) + (size_t)(2 * nmax + N) * sizeof(int) + 32;
    const size_t psi_bytes = (size_t)N * (nmax + 1) * sizeof(cplx);
    const int stage_psi = smem + psi_bytes <= 100 * 1024;       // two CTAs per SM at least; larger walkers are read from global
    if (stage_psi) smem += psi_bytes;
    cudaError_t e = func_config(c, (const void*)k_reference, 128, smem, nullptr);
    if (e != cudaSuccess) return e;
    int64_t wpad = (nw + MSD_WT - 1) / MSD_WT * MSD_WT;
    dim3 grid((unsigned)wpad, 2);
    k_reference<<<grid, 128, smem, st>>>(N, ldN, sa, sb, nw, phi_a, phi_b, ws.theta[0], ws.theta[1],
                                         want_thetaT ? ws.thetaT[0] : nullptr, want_thetaT ? ws.thetaT[1] : nullptr,
                                         ws.det0, ws.g[0], ws.g[1], ws.wflags, stage_psi);
    return cudaGetLastError();
}

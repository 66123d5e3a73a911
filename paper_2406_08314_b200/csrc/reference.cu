// S1 "reference" (Wick step W1): per (walker, spin)
//   O0 = psi[occ_ref,:]  (Psi_T^+ phi of PAPER.md Eq. 13 for the reference determinant), row-pivoted Gauss-Jordan inverse,
//   det0 = det O0 (Eq. 13), Theta = psi O0^-1 (N x n), so that the reference Green's function of Eq. 14
//   is G0[occ_ref[l], q] = Theta[q, l]; active slice g[h, p] = Theta[p, pos(h)].
// One CTA per (walker, spin).  complex128 throughout.
#include "msd_internal.cuh"

__global__ void __launch_bounds__(256)
k_reference(int N, int ldN, SpinDev sa, SpinDev sb, int64_t nw, const cplx* __restrict__ phi_a,
            const cplx* __restrict__ phi_b, cplx* theta_a, cplx* theta_b, double* thetaT_a, double* thetaT_b,
            cplx* det0, cplx* g_a, cplx* g_b, int* wflags, int stage_psi, double* kappa2)
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
        if (kappa2 && tid == 0) kappa2[w * 2 + s] = 0.0;
        return;
    }
    cplx* lu = reinterpret_cast<cplx*>(smem_raw);          // [n][n]
    cplx* inv = lu + n * n;                                 // [n][n]
    int* piv = reinterpret_cast<int*>(inv + n * n);         // [n]
    int* vmap = piv + n;                                    // [N]  orbital -> active-virtual index or -1
    int* omap = vmap + N;                                   // [n]  position in occ_ref -> active-occupied index or -1
    int* csrc = omap + n;                                   // [n]  column permutation of the inverse
    const size_t ints_end = (((size_t)2 * n * n * sizeof(cplx) + (size_t)(3 * n + N) * sizeof(int)) + 15) / 16 * 16;
    cplx* fcol = reinterpret_cast<cplx*>(smem_raw + ints_end);      // [n]  column j before elimination step j
    // the walker block itself, rows padded to n + 1 complex (conflict-free column walks in the Theta product);
    // read once, coalesced -- the strided global reads psi[q*n + m] were the whole cost of this kernel
    const int lps = n + 1;
    cplx* psis = fcol + n;
    __shared__ int s_p;
    __shared__ int s_sing;
    __shared__ double s_sign;
    __shared__ double s_nrm[2];            // sum |O0|^2, sum |O0^-1|^2  (kappa2 = their product: conditioning of the reference block)

    for (int q = tid; q < N; q += nt) vmap[q] = -1;
    for (int l = tid; l < n; l += nt) { omap[l] = -1; piv[l] = l; }
    if (tid == 0) { s_sing = 0; s_sign = 1.0; s_nrm[0] = 0.0; s_nrm[1] = 0.0; }
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
    if (kappa2) {
        double v = 0.0;
        for (int e = tid; e < n * n; e += nt) v += cabs2(lu[e]);
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if ((tid & 31) == 0) atomicAdd(&s_nrm[0], v);
    }

    // --- in-place Gauss-Jordan inverse with partial pivoting (rows), in shared memory: every step updates all n x n entries
    //     with the whole CTA (an LU followed by per-column substitutions left all but n threads idle for half of the kernel).
    //     The pivots are those of the LU, so det0 = sign x product of pivots is unchanged. ---
    cplx d0 = cmake(1.0, 0.0);                              // thread 0: product of the pivots
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
            if (tid == 0) s_sign = -s_sign;
        }
        if (tid == 0) piv[j] = p;
        __syncthreads();
        const cplx pv = lu[j * n + j];
        const cplx rinv = cinv(pv);
        if (tid == 0) d0 = cmul(d0, pv);
        for (int i = tid; i < n; i += nt) fcol[i] = lu[i * n + j];
        __syncthreads();                                    // pv and column j are read by everyone before they change
        for (int c = tid; c < n; c += nt) lu[j * n + c] = cmul(c == j ? cmake(1.0, 0.0) : lu[j * n + c], rinv);
        __syncthreads();
        for (int e = tid; e < n * n; e += nt) {
            const int i = e / n, c = e - i * n;
            if (i == j) continue;
            const cplx v = (c == j) ? cmake(0.0, 0.0) : lu[e];
            lu[e] = cfms(fcol[i], lu[j * n + c], v);
        }
        __syncthreads();
    }
    const bool sing = s_sing != 0;
    if (tid == 0) {
        cplx d = sing ? cmake(0.0, 0.0) : cscale(s_sign, d0);
        det0[w * 2 + s] = d;
        if (sing) atomicOr(&wflags[w], 1);
        // (P O0)^-1 = O0^-1 P^-1: undo the row swaps on the columns, last swap first
        for (int c = 0; c < n; c++) csrc[c] = c;
        if (!sing)
            for (int j = n - 1; j >= 0; j--) { const int pj = piv[j]; const int t = csrc[j]; csrc[j] = csrc[pj]; csrc[pj] = t; }
    }
    __syncthreads();
    if (!sing) {
        double v = 0.0;
        for (int e = tid; e < n * n; e += nt) { const cplx t = lu[(e / n) * n + csrc[e % n]]; inv[e] = t; v += cabs2(t); }
        if (kappa2) {
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if ((tid & 31) == 0) atomicAdd(&s_nrm[1], v);
        }
    }
    __syncthreads();
    if (kappa2 && tid == 0) kappa2[w * 2 + s] = (n == 0) ? 0.0 : (sing ? __longlong_as_double(0x7ff0000000000000LL) : s_nrm[0] * s_nrm[1]);
    // --- Theta = psi O0^-1 and its three layouts ---
    const double nanv = __longlong_as_double(0x7ff8000000000000LL);
    // four outputs per thread at a time: four independent FMA chains (one chain of n complex FMAs per output is pure latency)
    for (int e0 = tid; e0 < N * n; e0 += 4 * nt) {
        int l[4], q[4];
        cplx acc[4];
#pragma unroll
        for (int u = 0; u < 4; u++) {
            const int e = min(e0 + u * nt, N * n - 1);     // clamped duplicates are computed and not stored
            l[u] = e / N; q[u] = e - l[u] * N;             // consecutive threads -> consecutive q
            acc[u] = cmake(0.0, 0.0);
        }
        if (sing) {
#pragma unroll
            for (int u = 0; u < 4; u++) acc[u] = cmake(nanv, nanv);
        } else if (stage_psi) {
            for (int m = 0; m < n; m++) {
#pragma unroll
                for (int u = 0; u < 4; u++) acc[u] = cfma(psis[q[u] * lps + m], inv[m * n + l[u]], acc[u]);
            }
        } else {
            for (int m = 0; m < n; m++) {
#pragma unroll
                for (int u = 0; u < 4; u++) acc[u] = cfma(psi[(int64_t)q[u] * n + m], inv[m * n + l[u]], acc[u]);
            }
        }
#pragma unroll
        for (int u = 0; u < 4; u++) {
            if (e0 + u * nt >= N * n) break;
            theta[(int64_t)q[u] * n + l[u]] = acc[u];
            if (thetaT) {
                double* tt = thetaT + ((w * n + l[u]) * 2) * (int64_t)ldN;     // rows (w, l, re/im), K = q contiguous
                tt[q[u]] = acc[u].x; tt[ldN + q[u]] = acc[u].y;
                if (q[u] == 0 && ldN > N) { tt[N] = 0.0; tt[ldN + N] = 0.0; }     // zero the even-stride pad
            }
            int r = vmap[q[u]], h = omap[l[u]];
            if (r >= 0 && h >= 0) g[(int64_t)(r * sp.n_o + h) * MSD_WT] = acc[u];
        }
    }
}

cudaError_t launch_reference(msd_ctx* c, int N, int ldN, SpinDev sa, SpinDev sb, int64_t nw, const cplx* phi_a,
                             const cplx* phi_b, Workspace& ws, bool want_thetaT, cudaStream_t st)
{
    int nmax = sa.n > sb.n ? sa.n : sb.n;
    size_t smem = (size_t)2 * nmax * nmax * sizeof(cplx) + (size_t)(3 * nmax + N) * sizeof(int) + 32 + (size_t)nmax * sizeof(cplx);
    const size_t psi_bytes = (size_t)N * (nmax + 1) * sizeof(cplx);
    const int stage_psi = smem + psi_bytes <= 100 * 1024;       // two CTAs per SM at least; larger walkers are read from global
    if (stage_psi) smem += psi_bytes;
    cudaError_t e = func_config(c, (const void*)k_reference, 256, smem, nullptr);
    if (e != cudaSuccess) return e;
    int64_t wpad = (nw + MSD_WT - 1) / MSD_WT * MSD_WT;
    dim3 grid((unsigned)wpad, 2);
    k_reference<<<grid, 256, smem, st>>>(N, ldN, sa, sb, nw, phi_a, phi_b, ws.theta[0], ws.theta[1],
                                         want_thetaT ? ws.thetaT[0] : nullptr, want_thetaT ? ws.thetaT[1] : nullptr,
                                         ws.det0, ws.g[0], ws.g[1], ws.wflags, stage_psi, ws.kappa2);
    return cudaGetLastError();
}

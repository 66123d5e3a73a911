// One phaseless-AFQMC propagation step around the hot path (Eq. 5, Eq. 7-12).
//   h'      = h - 1/2 sum_g L^g L^g                                             Eq. 4
//   xbar_g  = -i sqrt(dt) v_g,  v = the force bias of msd_force_bias            Eq. 7 (reading A20: the factor i)
//   B(y)    = exp(-dt h'/2) exp(i sqrt(dt) sum_g y_g L^g) exp(-dt h'/2)         Eq. 5 (A20), y = x - xbar
//   psi'    = B(x - xbar) psi ;  S = <Psi_T|psi'>/<Psi_T|psi> ; theta = arg S   Eq. 8-9
//   I       = S exp(x.xbar - xbar.xbar/2) ;  I_ph = |I| max(0, cos theta) ;  w' = I_ph w      Eq. 10-12
// exp(-dt h'/2) is built once per time step size by scaling and squaring (Taylor order 16 of the scaled matrix) with the
// library's own FP64 DMMA GEMM; the field exponential is applied as a Taylor series of order n_taylor (reading A21).
// The field matrices A_w = i sqrt(dt) sum_g y_g L^g of all walkers are ONE dense contraction of L with the shifted fields
// (N^2 x n_chol by n_chol x 2 n_w) -> DMMA GEMM; the orbital update of a walker is a chain of small products -> one CTA.
#include "msd_internal.cuh"
#include <cmath>

// LT[(p, q)][g] = L[g][p][q]  (g contiguous, row stride ldg even): the A operand of the field-matrix GEMM
__global__ void k_prop_lt(const double* __restrict__ L, int n_chol, int NN, int ldg, double* __restrict__ LT)
{
    __shared__ double tile[32][33];
    const int g0 = blockIdx.y * 32, m0 = blockIdx.x * 32;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int g = g0 + r, m = m0 + threadIdx.x;
        tile[r][threadIdx.x] = (g < n_chol && m < NN) ? L[(int64_t)g * NN + m] : 0.0;
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int m = m0 + r, g = g0 + threadIdx.x;
        if (m < NN && g < ldg) LT[(int64_t)m * ldg + g] = tile[threadIdx.x][r];
    }
}

// out = alpha * A + beta * I   (n x n, row stride ld)
__global__ void k_prop_axpi(int n, int ld, double alpha, const double* __restrict__ A, double beta, double* __restrict__ out)
{
    const int i = blockIdx.y, j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= ld) return;
    out[(int64_t)i * ld + j] = (j < n) ? alpha * A[(int64_t)i * ld + j] + ((i == j) ? beta : 0.0) : 0.0;
}

// h' = h - 1/2 S,  S = sum_g L^g L^g accumulated by the GEMM into S (row stride ld)
__global__ void k_prop_hprime(int n, int ld, const double* __restrict__ h1, const double* __restrict__ S, double* __restrict__ hp)
{
    const int i = blockIdx.y, j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= ld) return;
    hp[(int64_t)i * ld + j] = (j < n) ? h1[(int64_t)i * n + j] - 0.5 * S[(int64_t)i * ld + j] : 0.0;
}

// Shifted fields as the B operand of the field-matrix GEMM, and the exponent of Eq. 10.  With xbar = -i sqrt(dt) v and
// y = x - xbar = x + i sqrt(dt) v:   A_w = i sqrt(dt) sum_g y_g L^g  has  Re A = -sqrt(dt) sum Im(y) L,  Im A = sqrt(dt) sum Re(y) L
//   Y[(w, 0)][g] = -sqrt(dt) Im y_g = -dt Re v_g ,   Y[(w, 1)][g] = sqrt(dt) Re y_g = sqrt(dt) x_g - dt Im v_g
//   expo[w] = x.xbar - xbar.xbar/2 = -i sqrt(dt) sum_g x_g v_g + dt/2 sum_g v_g^2          (plain sums, no conjugation)
__global__ void __launch_bounds__(256)
k_prop_fields(int n_chol, int ldg, double dt, const double* __restrict__ x, const cplx* __restrict__ v, double* __restrict__ Y,
              cplx* __restrict__ expo)
{
    const int64_t w = blockIdx.x;
    const double sq = sqrt(dt);
    cplx e = cmake(0.0, 0.0);
    for (int g = threadIdx.x; g < ldg; g += blockDim.x) {
        double y0 = 0.0, y1 = 0.0;
        if (g < n_chol) {
            const double xg = x[w * n_chol + g];
            const cplx vg = v[w * n_chol + g];
            y0 = -dt * vg.x;
            y1 = sq * xg - dt * vg.y;
            // -i sqrt(dt) x v = sqrt(dt) x (v_i, -v_r);   dt/2 v^2 = dt/2 (v_r^2 - v_i^2, 2 v_r v_i)
            e.x += sq * xg * vg.y + 0.5 * dt * (vg.x * vg.x - vg.y * vg.y);
            e.y += -sq * xg * vg.x + dt * vg.x * vg.y;
        }
        Y[(w * 2 + 0) * ldg + g] = y0;
        Y[(w * 2 + 1) * ldg + g] = y1;
    }
    __shared__ double red[2][8];
    for (int o = 16; o > 0; o >>= 1) { e.x += __shfl_down_sync(0xffffffffu, e.x, o); e.y += __shfl_down_sync(0xffffffffu, e.y, o); }
    if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = e.x; red[1][threadIdx.x >> 5] = e.y; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double sx = 0.0, sy = 0.0;
        for (int i = 0; i < (int)(blockDim.x >> 5); i++) { sx += red[0][i]; sy += red[1][i]; }
        expo[w] = cmake(sx, sy);
    }
}

// Orbital update of one (walker, spin):  psi <- E * taylor_n(A_w) * E * psi   (E real N x N, A_w complex N x N, psi N x n).
// The walker and the running Taylor term live in shared memory; a thread owns output elements (p, i) and streams row p of
// the left operand from global memory (L1: consecutive q of one thread share cache lines).
template <bool CPLX_LEFT>
__device__ __forceinline__ void prop_matmul(int N, int n, int ldl, const void* left, const cplx* __restrict__ src, cplx* __restrict__ dst,
                                            double scale)
{
    // four outputs per thread at a time -- column i of rows p, p + G, p + 2G, p + 3G (G = ceil(N / 4)): four independent FMA
    // chains (one chain of N complex FMAs per output is pure latency) that share every shared-memory read of src;
    // consecutive threads keep consecutive i (conflict-free shared memory, the row loads broadcast within a warp)
    const int G = (N + 3) >> 2;
    for (int e = threadIdx.x; e < G * n; e += blockDim.x) {
        const int p = e / n, i = e - p * n;
        int pr[4];
        cplx acc[4];
#pragma unroll
        for (int u = 0; u < 4; u++) { pr[u] = min(p + u * G, N - 1); acc[u] = cmake(0.0, 0.0); }     // clamped duplicates are not stored
        if (CPLX_LEFT) {
            const cplx* L_ = reinterpret_cast<const cplx*>(left);
#pragma unroll 2
            for (int q = 0; q < N; q++) {
                const cplx sv = src[q * n + i];
#pragma unroll
                for (int u = 0; u < 4; u++) acc[u] = cfma(__ldg(L_ + (int64_t)pr[u] * N + q), sv, acc[u]);
            }
        } else {
            const double* L_ = reinterpret_cast<const double*>(left);
#pragma unroll 2
            for (int q = 0; q < N; q++) {
                const cplx sv = src[q * n + i];
#pragma unroll
                for (int u = 0; u < 4; u++) {
                    const double a = __ldg(L_ + (int64_t)pr[u] * ldl + q);
                    acc[u].x = fma(a, sv.x, acc[u].x); acc[u].y = fma(a, sv.y, acc[u].y);
                }
            }
        }
#pragma unroll
        for (int u = 0; u < 4; u++)
            if (p + u * G < N) dst[(p + u * G) * n + i] = cscale(scale, acc[u]);
    }
}

// The same product on the FP64 tensor cores (DMMA m8n8k4) for n <= 8 NT columns: a warp owns two 8-row tiles of the result
// and all NT column tiles; per k-step of 4 it loads its two left-operand fragments from global memory (L1), the NT
// right-operand fragments from shared memory, and issues 4 (complex left) or 2 (real left) DMMAs per tile:
//   Cr += Ar Xr - Ai Xi,  Ci += Ar Xi + Ai Xr.
template <bool CPLX_LEFT, int NT>
__device__ __forceinline__ void prop_matmul_mma(int N, int n, int ldl, const void* left, const cplx* __restrict__ src,
                                                cplx* __restrict__ dst, double scale)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int MT = (N + 7) >> 3;
    for (int mt0 = wid; mt0 < MT; mt0 += 2 * nwarp) {
        const int mt1 = mt0 + nwarp;
        const bool two = mt1 < MT;
        const int p0 = min(mt0 * 8 + g, N - 1), p1 = min(mt1 * 8 + g, N - 1);      // clamped rows are computed and not stored
        double cr[2][NT][2], ci[2][NT][2];
#pragma unroll
        for (int m = 0; m < 2; m++)
#pragma unroll
            for (int nt = 0; nt < NT; nt++) { cr[m][nt][0] = cr[m][nt][1] = 0.0; ci[m][nt][0] = ci[m][nt][1] = 0.0; }
        for (int q0 = 0; q0 < N; q0 += 4) {
            const int q = q0 + t;
            const bool qok = q < N;
            double ar[2], ai[2];
            if (CPLX_LEFT) {
                const cplx* L_ = reinterpret_cast<const cplx*>(left);
                const cplx a0 = qok ? __ldg(L_ + (int64_t)p0 * N + q) : cmake(0.0, 0.0);
                const cplx a1 = (qok && two) ? __ldg(L_ + (int64_t)p1 * N + q) : cmake(0.0, 0.0);
                ar[0] = a0.x; ai[0] = a0.y; ar[1] = a1.x; ai[1] = a1.y;
            } else {
                const double* L_ = reinterpret_cast<const double*>(left);
                ar[0] = qok ? __ldg(L_ + (int64_t)p0 * ldl + q) : 0.0;
                ar[1] = (qok && two) ? __ldg(L_ + (int64_t)p1 * ldl + q) : 0.0;
                ai[0] = ai[1] = 0.0;
            }
#pragma unroll
            for (int nt = 0; nt < NT; nt++) {
                const int i = nt * 8 + g;
                const cplx x = (qok && i < n) ? src[q * n + i] : cmake(0.0, 0.0);
#pragma unroll
                for (int m = 0; m < 2; m++) {
                    if (m == 1 && !two) continue;        // warp-uniform
                    dmma884(cr[m][nt][0], cr[m][nt][1], ar[m], x.x);
                    dmma884(ci[m][nt][0], ci[m][nt][1], ar[m], x.y);
                    if (CPLX_LEFT) {
                        dmma884(cr[m][nt][0], cr[m][nt][1], -ai[m], x.y);
                        dmma884(ci[m][nt][0], ci[m][nt][1], ai[m], x.x);
                    }
                }
            }
        }
#pragma unroll
        for (int m = 0; m < 2; m++) {
            const int row = (m ? mt1 : mt0) * 8 + g;
            if ((m == 1 && !two) || row >= N) continue;
#pragma unroll
            for (int nt = 0; nt < NT; nt++)
#pragma unroll
                for (int k = 0; k < 2; k++) {
                    const int col = nt * 8 + 2 * t + k;
                    if (col < n) dst[row * n + col] = cmake(scale * cr[m][nt][k], scale * ci[m][nt][k]);
                }
        }
    }
}

// dispatch: tensor-core form for n <= 32, the scalar form beyond
template <bool CPLX_LEFT>
__device__ __forceinline__ void prop_product(int N, int n, int ldl, const void* left, const cplx* __restrict__ src,
                                             cplx* __restrict__ dst, double scale)
{
    if (n <= 8) prop_matmul_mma<CPLX_LEFT, 1>(N, n, ldl, left, src, dst, scale);
    else if (n <= 16) prop_matmul_mma<CPLX_LEFT, 2>(N, n, ldl, left, src, dst, scale);
    else if (n <= 24) prop_matmul_mma<CPLX_LEFT, 3>(N, n, ldl, left, src, dst, scale);
    else if (n <= 32) prop_matmul_mma<CPLX_LEFT, 4>(N, n, ldl, left, src, dst, scale);
    else prop_matmul<CPLX_LEFT>(N, n, ldl, left, src, dst, scale);
}

__global__ void __launch_bounds__(256)
k_prop_orbitals(int N, int ldN, int na, int nb, int n_taylor, const double* __restrict__ E, const cplx* __restrict__ Aw,
                cplx* phi_a, cplx* phi_b)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int s = blockIdx.y;
    const int64_t w = blockIdx.x;
    const int n = s ? nb : na;
    if (n == 0) return;
    cplx* phi = (s ? phi_b : phi_a) + w * (int64_t)N * n;
    const cplx* A = Aw + w * (int64_t)N * N;
    cplx* t0 = reinterpret_cast<cplx*>(smem_raw);       // running term
    cplx* t1 = t0 + N * n;                               // next term
    cplx* sum = t1 + N * n;                              // partial sum of the series
    for (int e = threadIdx.x; e < N * n; e += blockDim.x) t1[e] = phi[e];
    __syncthreads();
    prop_product<false>(N, n, ldN, E, t1, t0, 1.0);      // t0 = E psi
    __syncthreads();
    for (int e = threadIdx.x; e < N * n; e += blockDim.x) sum[e] = t0[e];
    __syncthreads();
    for (int k = 1; k <= n_taylor; k++) {
        prop_product<true>(N, n, 0, A, t0, t1, 1.0 / (double)k);      // term_k = A term_{k-1} / k
        __syncthreads();
        for (int e = threadIdx.x; e < N * n; e += blockDim.x) { sum[e] = cadd(sum[e], t1[e]); }
        cplx* tmp = t0; t0 = t1; t1 = tmp;
        __syncthreads();
    }
    prop_product<false>(N, n, ldN, E, sum, t1, 1.0);     // psi' = E sum
    __syncthreads();
    for (int e = threadIdx.x; e < N * n; e += blockDim.x) phi[e] = t1[e];
}

// Eq. 8-12 per walker.  out[w][8] = (Re S, Im S, theta, I_ph, Re ovlp', Im ovlp', Re I, Im I); weights updated in place.
__global__ void k_prop_finish(int64_t nw, const cplx* __restrict__ ov_old, const cplx* __restrict__ ov_new,
                              const cplx* __restrict__ expo, double* weights, double* out, const int* __restrict__ fl_old,
                              int* flags)
{
    const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= nw) return;
    const cplx S = cdiv(ov_new[w], ov_old[w]);
    const double theta = atan2(S.y, S.x);
    const double m = exp(expo[w].x);
    const cplx ph = cmake(m * cos(expo[w].y), m * sin(expo[w].y));
    const cplx I = cmul(S, ph);
    const double c = cos(theta);
    const double Iph = sqrt(cabs2(I)) * (c > 0.0 ? c : 0.0);
    double* o = out + w * 8;
    o[0] = S.x; o[1] = S.y; o[2] = theta; o[3] = Iph; o[4] = ov_new[w].x; o[5] = ov_new[w].y; o[6] = I.x; o[7] = I.y;
    if (weights) weights[w] *= Iph;
    if (flags) flags[w] = (fl_old ? fl_old[w] : 0) | flags[w];
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
static cudaError_t real_gemm_nn_sym(msd_ctx* c, int n, int ld, const double* A, const double* B, double* C, cudaStream_t st)
{
    // C = A * B for SYMMETRIC B (B^T = B), all n x n with row stride ld (even): the library's TN kernel computes A B^T
    GemmArgs a;
    a.A = A; a.B = B; a.C = C;
    a.M = n; a.N = ld; a.K = ld;
    a.lda = ld; a.ldb = ld; a.strideA = 0; a.strideB = 0; a.batch = 1;
    a.zdiv = 1; a.strideC_hi = 0; a.strideC_lo = 0; a.cs_m = ld / 2; a.cs_j = 1;
    a.accumulate = 0;
    cudaError_t e = launch_gemm_tn(c, a, st);
    c->launches++;
    return e;
}

// builds LT, h' (once) and E = exp(-dt h'/2); h1, L are HOST arrays (the ones msd_setup was given)
cudaError_t prop_setup(msd_ctx* c, double dt, int n_taylor, const double* h1, const double* L, cudaStream_t st)
{
    const int N = c->N, ld = N + (N & 1), ng = c->n_chol, ldg = ng + (ng & 1);
    cudaError_t e;
    if (!c->d_LT) {
        double* d_L = nullptr; double* d_h1 = nullptr; double* d_S = nullptr; double* d_Ld = nullptr;
        // L twice: dense [g][p][q] (source of LT) and with row stride ld (even) for the GEMM (one spare row: an odd N reads it)
        if ((e = cudaMalloc(&d_Ld, sizeof(double) * (size_t)ng * N * N)) != cudaSuccess) return e;
        if ((e = cudaMalloc(&d_L, sizeof(double) * ((size_t)ng * N + 1) * ld)) != cudaSuccess) return e;
        if ((e = cudaMalloc(&d_h1, sizeof(double) * (size_t)N * N)) != cudaSuccess) return e;
        if ((e = cudaMalloc(&d_S, sizeof(double) * (size_t)ld * ld)) != cudaSuccess) return e;
        if ((e = cudaMalloc(&c->d_LT, sizeof(double) * (size_t)N * N * ldg)) != cudaSuccess) return e;
        if ((e = cudaMalloc(&c->d_hp, sizeof(double) * (size_t)ld * ld)) != cudaSuccess) return e;
        if ((e = cudaMalloc(&c->d_E, sizeof(double) * (size_t)ld * ld * 3)) != cudaSuccess) return e;
        cudaMemsetAsync(c->d_hp, 0, sizeof(double) * (size_t)ld * ld, st);
        cudaMemsetAsync(c->d_E, 0, sizeof(double) * (size_t)ld * ld * 3, st);
        cudaMemcpyAsync(d_Ld, L, sizeof(double) * (size_t)ng * N * N, cudaMemcpyHostToDevice, st);
        cudaMemcpyAsync(d_h1, h1, sizeof(double) * (size_t)N * N, cudaMemcpyHostToDevice, st);
        cudaMemsetAsync(d_L, 0, sizeof(double) * ((size_t)ng * N + 1) * ld, st);
        cudaMemcpy2DAsync(d_L, ld * sizeof(double), d_Ld, N * sizeof(double), N * sizeof(double), (size_t)ng * N,
                          cudaMemcpyDeviceToDevice, st);
        {
            dim3 grid((N * N + 31) / 32, (ldg + 31) / 32), blk(32, 8);
            k_prop_lt<<<grid, blk, 0, st>>>(d_Ld, ng, N * N, ldg, c->d_LT);
            c->launches++;
        }
        // S = sum_g L^g L^g : batch over g, partial products meet in RED.ADD.F64
        cudaMemsetAsync(d_S, 0, sizeof(double) * (size_t)ld * ld, st);
        GemmArgs a;
        a.A = d_L; a.B = d_L; a.C = d_S;
        a.M = N; a.N = ld; a.K = ld; a.lda = ld; a.ldb = ld;
        a.strideA = (int64_t)N * ld; a.strideB = (int64_t)N * ld; a.batch = ng;
        a.zdiv = 1; a.strideC_hi = 0; a.strideC_lo = 0; a.cs_m = ld / 2; a.cs_j = 1;
        a.accumulate = 2;
        if ((e = launch_gemm_tn(c, a, st)) != cudaSuccess) return e;
        c->launches++;
        k_prop_hprime<<<dim3((ld + 127) / 128, N), 128, 0, st>>>(N, ld, d_h1, d_S, c->d_hp);
        c->launches++;
        if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return e;
        cudaFree(d_L); cudaFree(d_h1); cudaFree(d_S); cudaFree(d_Ld);
    }
    // E = exp(M), M = -dt/2 h': scale by 2^-s so that the 1-norm is <= 1/2, Taylor order 16 by Horner, square s times
    std::vector<double> hp((size_t)N * ld);
    if ((e = cudaMemcpyAsync(hp.data(), c->d_hp, sizeof(double) * (size_t)N * ld, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return e;
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return e;
    double nrm = 0.0;
    for (int j = 0; j < N; j++) { double s = 0.0; for (int i = 0; i < N; i++) s += fabs(hp[(size_t)i * ld + j]); nrm = std::max(nrm, s); }
    nrm *= 0.5 * fabs(dt);
    int sq = 0;
    while (nrm > 0.5 && sq < 60) { nrm *= 0.5; sq++; }
    double* X = c->d_E + (size_t)ld * ld;          // scaled matrix
    double* T = c->d_E + (size_t)2 * ld * ld;      // scratch
    double* Ecur = c->d_E;
    const dim3 eg((ld + 127) / 128, N);
    k_prop_axpi<<<eg, 128, 0, st>>>(N, ld, -0.5 * dt / std::ldexp(1.0, sq), c->d_hp, 0.0, X);
    constexpr int ORDER = 16;
    // Horner: P = I + X/ORDER; for k = ORDER-1 .. 1: P = I + (X P)/k
    k_prop_axpi<<<eg, 128, 0, st>>>(N, ld, 1.0 / ORDER, X, 1.0, Ecur);
    c->launches += 2;
    for (int k = ORDER - 1; k >= 1; k--) {
        if ((e = real_gemm_nn_sym(c, N, ld, X, Ecur, T, st)) != cudaSuccess) return e;      // X P (P is a polynomial in X: symmetric)
        k_prop_axpi<<<eg, 128, 0, st>>>(N, ld, 1.0 / k, T, 1.0, Ecur);
        c->launches++;
    }
    for (int i = 0; i < sq; i++) {
        if ((e = real_gemm_nn_sym(c, N, ld, Ecur, Ecur, T, st)) != cudaSuccess) return e;
        k_prop_axpi<<<eg, 128, 0, st>>>(N, ld, 1.0, T, 0.0, Ecur);
        c->launches++;
    }
    c->prop_dt = dt; c->prop_taylor = n_taylor;
    return cudaStreamSynchronize(st);
}

cudaError_t launch_prop_fields(msd_ctx* c, int64_t nw, const double* x, const cplx* v, double* Y, cplx* expo, cudaStream_t st)
{
    const int ng = c->n_chol, ldg = ng + (ng & 1);
    k_prop_fields<<<(unsigned)nw, 256, 0, st>>>(ng, ldg, c->prop_dt, x, v, Y, expo);
    c->launches++;
    return cudaGetLastError();
}

// A_w[p][q] for all walkers of the chunk: (N^2 x n_chol) times (n_chol x 2 n_w), FP64 DMMA
cudaError_t launch_prop_vhs(msd_ctx* c, int64_t nw, const double* Y, cplx* Aw, cudaStream_t st)
{
    const int N = c->N, ng = c->n_chol, ldg = ng + (ng & 1);
    GemmArgs a;
    a.A = c->d_LT; a.B = Y; a.C = reinterpret_cast<double*>(Aw);
    a.M = N * N; a.N = (int)(2 * nw); a.K = ldg;
    a.lda = ldg; a.ldb = ldg; a.strideA = 0; a.strideB = 0; a.batch = 1;
    a.zdiv = 1; a.strideC_hi = 0; a.strideC_lo = 0; a.cs_m = 1; a.cs_j = (int64_t)N * N;
    a.accumulate = 0;
    cudaError_t e = launch_gemm_tn(c, a, st);
    c->launches++;
    return e;
}

cudaError_t launch_prop_orbitals(msd_ctx* c, int64_t nw, const cplx* Aw, cplx* phi_a, cplx* phi_b, cudaStream_t st)
{
    const int N = c->N, ld = N + (N & 1);
    const int nmax = std::max(c->sp[0].n, c->sp[1].n);
    const size_t smem = (size_t)3 * N * nmax * sizeof(cplx);
    cudaError_t e = func_config(c, (const void*)k_prop_orbitals, 256, smem, nullptr);
    if (e != cudaSuccess) return e;
    k_prop_orbitals<<<dim3((unsigned)nw, 2), 256, smem, st>>>(N, ld, c->sp[0].n, c->sp[1].n, c->prop_taylor, c->d_E, Aw, phi_a, phi_b);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_prop_finish(msd_ctx* c, int64_t nw, const cplx* ov_old, const cplx* ov_new, const cplx* expo, double* weights,
                               double* out, const int* fl_old, int* flags, cudaStream_t st)
{
    k_prop_finish<<<(unsigned)((nw + 127) / 128), 128, 0, st>>>(nw, ov_old, ov_new, expo, weights, out, fl_old, flags);
    c->launches++;
    return cudaGetLastError();
}

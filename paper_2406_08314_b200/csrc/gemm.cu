// FP64 tensor-core (DMMA, mma.sync.m8n8k4.f64) batched GEMM used by the dense contractions of the path:
//   S6 force bias   fb[g][w]   = sum_(r,q) L_sub[g][(r,q)] G[w][(r,q)]          (Eq. 7)
//   S7 Lambda       Lam[(g,r)][(w,i)] = sum_q L_sub[(g,r)][q] Theta_w[q][i]     (half rotation)
//   S7 V            V_w[x][y]  = sum_g B_w[x][g] B'_w[y][g]                      (two-body tensor in the active window)
// All three are  C[m][n] (+)= sum_k A[m][k] B[n][k]  with both operands K-contiguous ("TN"), real FP64;
// complex operands are expressed as real ones by the callers (see dense.cu).
//
// tcgen05/UMMA has no f64 kind, so FP64 tensor work on sm_100a goes through warp-level mma.sync; the bench-side probe
// (csrc/probes.cu) measured 37.1 TFLOP/s for DMMA and 36.3 for DFMA on B200 (they share the FP64 units).
// Tiles: CTA BM x BN x 16, 3-stage cp.async ring, warp tile 32 x 32 (4 x 4 DMMA tiles), fragments read from
// shared memory with row stride 20 doubles (conflict-free for the 8x4 fragment pattern).
#include "msd_internal.cuh"

#define BK 16
#define LDS_ 20       // BK + 4
#define STAGES 3

template <int BM, int BN, int WARPS_M, int WARPS_N, bool BX>
__global__ void __launch_bounds__(WARPS_M * WARPS_N * 32)
k_gemm_tn(GemmArgs g)
{
    constexpr int NT = WARPS_M * WARPS_N * 32;
    constexpr int WM = BM / WARPS_M, WN = BN / WARPS_N;       // warp tile
    constexpr int TM = WM / 8, TN = WN / 8;
    extern __shared__ __align__(16) double smem_gemm[];
    double* As = smem_gemm;                                    // [STAGES][BM][LDS_]
    constexpr int BROWS = BX ? BN / 2 : BN;                    // expand mode stages BN/2 complex rows
    double* Bs = smem_gemm + STAGES * BM * LDS_;               // [STAGES][BROWS][LDS_]
    const int z = blockIdx.z / g.ksplit, ks = blockIdx.z - z * g.ksplit;
    if (g.sel) { const bool hi = !(g.sel[2 * z] <= g.sel_thr) || !(g.sel[2 * z + 1] <= g.sel_thr); if (hi != (g.sel_hi != 0)) return; }
    if (g.symmetric && (int)(blockIdx.x * BN + BN) / 2 - 1 < (int)(blockIdx.y * BM)) return;   // strictly lower tile
    const double* A = g.A + (int64_t)z * g.strideA;
    const double* B = g.B + (int64_t)z * g.strideB;
    const int m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int wm = (wid % WARPS_M) * WM, wn = (wid / WARPS_M) * WN;
    const int gq = lane >> 2, tq = lane & 3;
    const int KT_all = (g.K + BK - 1) / BK;
    const int kt_per = (KT_all + g.ksplit - 1) / g.ksplit;
    const int kt_begin = ks * kt_per;
    const int KT = min(kt_per, KT_all - kt_begin);             // k-tiles of this split (may be <= 0 for the last)
    if (KT <= 0) return;

    auto load_tile = [&](int stage, int kt) {
        const int k0 = (kt_begin + kt) * BK;
        double* as = As + stage * BM * LDS_;
        double* bs = Bs + stage * BROWS * LDS_;
        for (int c = tid; c < BM * (BK / 2); c += NT) {
            int r = c / (BK / 2), kc = (c % (BK / 2)) * 2;
            int m = m0 + r, k = k0 + kc;
            bool ok = (m < g.M) && (k < g.K);
            const double* src = ok ? (A + (int64_t)m * g.lda + k) : A;
            cp_async16(as + r * LDS_ + kc, src, ok ? 16 : 0);
        }
        if (BX) {              // BN/2 complex rows: real column n = 2y + c is read from row y at fragment time
            for (int c = tid; c < (BN / 2) * (BK / 2); c += NT) {
                int r = c / (BK / 2), kc = (c % (BK / 2)) * 2;
                int y = n0 / 2 + r, k = k0 + kc;
                bool ok = (2 * y < g.N) && (k < g.K);
                const double* src = ok ? (B + (int64_t)y * g.ldb + k) : B;
                cp_async16(bs + r * LDS_ + kc, src, ok ? 16 : 0);
            }
        } else
        for (int c = tid; c < BN * (BK / 2); c += NT) {
            int r = c / (BK / 2), kc = (c % (BK / 2)) * 2;
            int n = n0 + r, k = k0 + kc;
            bool ok = (n < g.N) && (k < g.K);
            const double* src = ok ? (B + (int64_t)n * g.ldb + k) : B;
            cp_async16(bs + r * LDS_ + kc, src, ok ? 16 : 0);
        }
    };

    double acc[TM][TN][2];
#pragma unroll
    for (int i = 0; i < TM; i++)
#pragma unroll
        for (int j = 0; j < TN; j++) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }

    for (int s = 0; s < STAGES - 1; s++) {
        if (s < KT) load_tile(s, s);
        cp_async_commit();
    }
    for (int kt = 0; kt < KT; kt++) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        {
            int nk = kt + STAGES - 1;
            if (nk < KT) load_tile(nk % STAGES, nk);
            cp_async_commit();
        }
        const double* as = As + (kt % STAGES) * BM * LDS_ + (wm + gq) * LDS_ + tq;
        // bexpand: B[2y + c][2 gam + c'] = component (c ^ c') of the complex B[y][gam], negated for (c, c') = (0, 1);
        // c = gq & 1 and c' = tq & 1 are per-lane constants (warp and tile offsets are even)
        const double* bs = BX ? Bs + (kt % STAGES) * BROWS * LDS_ + ((wn + gq) >> 1) * LDS_ + ((tq & 2) | ((tq ^ gq) & 1))
                                     : Bs + (kt % STAGES) * BROWS * LDS_ + (wn + gq) * LDS_ + tq;
        constexpr int brow = BX ? 4 * LDS_ : 8 * LDS_;
        const long long bsign = (BX && !(gq & 1) && (tq & 1)) ? (long long)0x8000000000000000ull : 0ll;   // sign flip as an
        // integer XOR: a DADD/DMUL would take issue slots of the FP64 pipe that the DMMAs need
        auto kstep = [&](int kk) {
            double a[TM], b[TN];
#pragma unroll
            for (int i = 0; i < TM; i++) a[i] = as[i * 8 * LDS_ + kk * 4];
#pragma unroll
            for (int j = 0; j < TN; j++) { b[j] = bs[j * brow + kk * 4]; if (BX) b[j] = __longlong_as_double(__double_as_longlong(b[j]) ^ bsign); }
#pragma unroll
            for (int i = 0; i < TM; i++)
#pragma unroll
                for (int j = 0; j < TN; j++) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        };
        const int kleft = g.K - (kt_begin + kt) * BK;
        if (kleft >= BK) {
#pragma unroll
            for (int kk = 0; kk < BK / 4; kk++) kstep(kk);
        } else {               // short last k-tile (K = 100: 6 x 16 + 4): the zero-padded k-steps are skipped
#pragma unroll 1
            for (int kk = 0; kk < (kleft + 3) / 4; kk++) kstep(kk);
        }
    }
    cp_async_wait<0>();

    // epilogue: thread holds (row gq, columns 2 tq, 2 tq + 1) of every 8x8 tile = one complex / column pair
    double* Cz = g.C + 2 * ((int64_t)(z / g.zdiv) * g.strideC_hi + (int64_t)(z % g.zdiv) * g.strideC_lo);
#pragma unroll
    for (int i = 0; i < TM; i++) {
        const int m = m0 + wm + i * 8 + gq;
        if (m >= g.M) continue;
#pragma unroll
        for (int j = 0; j < TN; j++) {
            const int n = n0 + wn + j * 8 + 2 * tq;
            if (n >= g.N) continue;
            double2* dst = reinterpret_cast<double2*>(Cz + 2 * ((int64_t)m * g.cs_m + (int64_t)(n >> 1) * g.cs_j));
            double2 v = make_double2(acc[i][j][0], acc[i][j][1]);
            if (g.symmetric) {
                const int jc = n >> 1;
                if (jc < m) continue;
                *dst = v;
                if (jc > m)
                    *reinterpret_cast<double2*>(Cz + 2 * ((int64_t)jc * g.cs_m + (int64_t)m * g.cs_j)) = v;
                continue;
            }
            if (g.accumulate == 2) { atomicAdd(&dst->x, v.x); atomicAdd(&dst->y, v.y); continue; }
            if (g.accumulate) { double2 o = *dst; v.x += o.x; v.y += o.y; }
            *dst = v;
        }
    }
}

template <int BM, int BN, int WARPS_M, int WARPS_N, bool BX>
static cudaError_t launch_cfg_x(msd_ctx* c, const GemmArgs& a, cudaStream_t st)
{
    size_t smem = (size_t)STAGES * (BM + (BX ? BN / 2 : BN)) * LDS_ * sizeof(double);
    cudaError_t e = func_config(c, (const void*)k_gemm_tn<BM, BN, WARPS_M, WARPS_N, BX>, WARPS_M * WARPS_N * 32, smem, nullptr);
    if (e != cudaSuccess) return e;
    dim3 grid((a.N + BN - 1) / BN, (a.M + BM - 1) / BM, a.batch * a.ksplit);
    k_gemm_tn<BM, BN, WARPS_M, WARPS_N, BX><<<grid, WARPS_M * WARPS_N * 32, smem, st>>>(a);
    return cudaGetLastError();
}

template <int BM, int BN, int WARPS_M, int WARPS_N>
static cudaError_t launch_cfg(msd_ctx* c, const GemmArgs& a, cudaStream_t st)
{
    return a.bexpand ? launch_cfg_x<BM, BN, WARPS_M, WARPS_N, true>(c, a, st) : launch_cfg_x<BM, BN, WARPS_M, WARPS_N, false>(c, a, st);
}

cudaError_t launch_gemm_tn(msd_ctx* c, const GemmArgs& a, cudaStream_t st)
{
    const int n_sm = c->n_sm;
    if (a.M <= 0 || a.N <= 0 || a.batch <= 0) return cudaSuccess;
    if ((a.N & 1) || (a.K & 1) || (a.lda & 1) || (a.ldb & 1) || (a.strideA & 1) || (a.strideB & 1))
        return cudaErrorInvalidValue;     // callers pad to even sizes (16-byte cp.async chunks)
    if (a.bexpand && ((a.N & 1) || (a.strideB & 1))) return cudaErrorInvalidValue;
    if (a.ksplit < 1 || (a.ksplit > 1 && a.accumulate != 2) || (a.symmetric && (a.N != 2 * a.M || a.accumulate)))
        return cudaErrorInvalidValue;
    // Tile shape by a wave model: time ~ waves x (CTAs per SM) x BM x BN, waves = ceil(computed tiles / (SMs x CTAs per SM)).
    // Padding (e.g. P = 225 rows against 64- or 128-row tiles) and the partly filled last wave are what it minimises.
    struct Cand { int bm, bn, occ; };
    // CTAs per SM from shared memory and registers; the expand mode stages half the B rows
    const Cand cands[3] = {{128, 64, 2}, {64, 64, a.bexpand ? 4 : 3}, {48, 96, a.bexpand ? 4 : 3}};
    int best = 0; double best_cost = 0.0;
    for (int i = 0; i < 3; i++) {
        const int tm = (a.M + cands[i].bm - 1) / cands[i].bm, tn = (a.N + cands[i].bn - 1) / cands[i].bn;
        int64_t tiles = 0;
        if (a.symmetric) {
            for (int y = 0; y < tm; y++)
                for (int x = 0; x < tn; x++)
                    if (!((x * cands[i].bn + cands[i].bn) / 2 - 1 < y * cands[i].bm)) tiles++;
        } else tiles = (int64_t)tm * tn;
        tiles *= (int64_t)a.batch * a.ksplit;
        const int64_t slots = (int64_t)n_sm * cands[i].occ;
        const double cost = (double)((tiles + slots - 1) / slots) * cands[i].occ * cands[i].bm * cands[i].bn;
        if (i == 0 || cost < best_cost * 0.97) { best = i; best_cost = cost; }     // ties go to the larger tile
    }
    if (best == 0) return launch_cfg<128, 64, 4, 2>(c, a, st);
    if (best == 1) return launch_cfg<64, 64, 2, 2>(c, a, st);
    return launch_cfg<48, 96, 2, 2>(c, a, st);
}

// ------------------------------------------------------------------------------------------------
// Complex bilinear batched product by the 3-multiplication (Karatsuba) scheme, for the V contractions:
//   C[x][y] = sum_g A[x][g] B[y][g]        A, B complex rows (re, im interleaved, g contiguous), no conjugation
//   P1 = sum a_r b_r,  P2 = sum a_i b_i,  P3 = sum (a_r + a_i)(b_r + b_i);   C_r = P1 - P2,  C_i = P3 - P1 - P2
// Three real DMMA products per complex output instead of four (the real form [a_r a_i] x [[b_r b_i], [-b_i b_r]] of
// k_gemm_tn's expand mode): 25 % fewer tensor-pipe cycles.  One 16-byte shared-memory read yields (a_r, a_i) of a fragment
// element, the sum a_r + a_i is one DADD (3.5 % of the pipe time of the 27 DMMAs it feeds).  The imaginary part is formed
// by subtraction: its rounding error is relative to |A||B| instead of |C_i| (bounded by 3 eps sum |a||b|, far inside the
// 1e-8 Ha energy tolerance).
// CTA tile 48 rows x 48 complex columns, 4 warps of 24 x 24 (3 x 3 DMMA tiles x 3 products = 27 accumulator tiles),
// k-tile of 8 gamma (128-byte rows), 4-stage cp.async ring, row stride 24 doubles (conflict-free 16-byte fragment reads).
// ------------------------------------------------------------------------------------------------
#define V3_BM 48
#define V3_BN 48
#define V3_BG 8          // gamma per k-tile
#define V3_LD 24         // doubles per staged row: 2 * V3_BG + 8
#define V3_STAGES 4

__global__ void __launch_bounds__(128, 3) k_vgemm3m(GemmArgs g)
{
    extern __shared__ __align__(16) double smem_v3[];
    double* As = smem_v3;                                     // [STAGES][48][LD]
    double* Bs = smem_v3 + V3_STAGES * V3_BM * V3_LD;         // [STAGES][48][LD]
    const int z = blockIdx.z;
    if (g.sel) { const bool hi = !(g.sel[2 * z] <= g.sel_thr) || !(g.sel[2 * z + 1] <= g.sel_thr); if (hi != (g.sel_hi != 0)) return; }
    const int bx = blockIdx.x, by = blockIdx.y;
    if (g.symmetric && bx < by) return;                       // strictly lower tile (square complex tiles)
    const int Nc = g.N / 2, ngam = g.K / 2;
    const double* A = g.A + (int64_t)z * g.strideA;
    const double* B = g.B + (int64_t)z * g.strideB;
    const int m0 = by * V3_BM, n0 = bx * V3_BN;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int wm = (wid & 1) * 24, wn = (wid >> 1) * 24;
    const int gq = lane >> 2, tq = lane & 3;
    const int KT = (ngam + V3_BG - 1) / V3_BG;

    auto load_tile = [&](int stage, int kt) {
        const int g0 = kt * V3_BG;
        double* as = As + stage * V3_BM * V3_LD;
        double* bs = Bs + stage * V3_BN * V3_LD;
        // 48 rows x 8 chunks of 16 bytes (one complex each) per operand; 128 threads: 3 chunks of A and 3 of B each
        for (int c = tid; c < V3_BM * V3_BG; c += 128) {
            const int r = c >> 3, kc = c & 7;
            const bool ok = (m0 + r < g.M) && (g0 + kc < ngam);
            cp_async16(as + r * V3_LD + 2 * kc, ok ? A + (int64_t)(m0 + r) * g.lda + 2 * (g0 + kc) : A, ok ? 16 : 0);
        }
        for (int c = tid; c < V3_BN * V3_BG; c += 128) {
            const int r = c >> 3, kc = c & 7;
            const bool ok = (n0 + r < Nc) && (g0 + kc < ngam);
            cp_async16(bs + r * V3_LD + 2 * kc, ok ? B + (int64_t)(n0 + r) * g.ldb + 2 * (g0 + kc) : B, ok ? 16 : 0);
        }
    };

    double p1[3][3][2], p2[3][3][2], p3[3][3][2];
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++)
#pragma unroll
            for (int t = 0; t < 2; t++) { p1[i][j][t] = 0.0; p2[i][j][t] = 0.0; p3[i][j][t] = 0.0; }

    for (int s = 0; s < V3_STAGES - 1; s++) {
        if (s < KT) load_tile(s, s);
        cp_async_commit();
    }
    for (int kt = 0; kt < KT; kt++) {
        cp_async_wait<V3_STAGES - 2>();
        __syncthreads();
        {
            const int nk = kt + V3_STAGES - 1;
            if (nk < KT) load_tile(nk % V3_STAGES, nk);
            cp_async_commit();
        }
        const double* as = As + (kt % V3_STAGES) * V3_BM * V3_LD + (wm + gq) * V3_LD + 2 * tq;
        const double* bs = Bs + (kt % V3_STAGES) * V3_BN * V3_LD + (wn + gq) * V3_LD + 2 * tq;
#pragma unroll
        for (int kk = 0; kk < V3_BG / 4; kk++) {
            double ar[3], ai[3], asum[3], br[3], bi[3], bsum[3];
#pragma unroll
            for (int i = 0; i < 3; i++) {
                const double2 v = *reinterpret_cast<const double2*>(as + i * 8 * V3_LD + kk * 8);
                ar[i] = v.x; ai[i] = v.y; asum[i] = v.x + v.y;
            }
#pragma unroll
            for (int j = 0; j < 3; j++) {
                const double2 v = *reinterpret_cast<const double2*>(bs + j * 8 * V3_LD + kk * 8);
                br[j] = v.x; bi[j] = v.y; bsum[j] = v.x + v.y;
            }
#pragma unroll
            for (int i = 0; i < 3; i++)
#pragma unroll
                for (int j = 0; j < 3; j++) {
                    dmma884(p1[i][j][0], p1[i][j][1], ar[i], br[j]);
                    dmma884(p2[i][j][0], p2[i][j][1], ai[i], bi[j]);
                    dmma884(p3[i][j][0], p3[i][j][1], asum[i], bsum[j]);
                }
        }
    }
    cp_async_wait<0>();

    // epilogue: thread holds rows m = m0 + wm + 8 i + gq, complex columns y = n0 + wn + 8 j + 2 tq (+1)
    double* Cz = g.C + 2 * ((int64_t)(z / g.zdiv) * g.strideC_hi + (int64_t)(z % g.zdiv) * g.strideC_lo);
#pragma unroll
    for (int i = 0; i < 3; i++) {
        const int m = m0 + wm + i * 8 + gq;
        if (m >= g.M) continue;
#pragma unroll
        for (int j = 0; j < 3; j++)
#pragma unroll
            for (int t = 0; t < 2; t++) {
                const int y = n0 + wn + j * 8 + 2 * tq + t;
                if (y >= Nc) continue;
                if (g.symmetric && y < m) continue;
                const double2 v = make_double2(p1[i][j][t] - p2[i][j][t], p3[i][j][t] - p1[i][j][t] - p2[i][j][t]);
                *reinterpret_cast<double2*>(Cz + 2 * ((int64_t)m * g.cs_m + (int64_t)y * g.cs_j)) = v;
                if (g.symmetric && y > m) *reinterpret_cast<double2*>(Cz + 2 * ((int64_t)y * g.cs_m + (int64_t)m * g.cs_j)) = v;
            }
    }
}

// A, B: complex rows (g.M rows of A, g.N / 2 rows of B), g.K = 2 x gammas doubles per row; C as in k_gemm_tn
cudaError_t launch_vgemm3m(msd_ctx* c, const GemmArgs& a, cudaStream_t st)
{
    if (a.M <= 0 || a.N <= 0 || a.batch <= 0) return cudaSuccess;
    if ((a.N & 1) || (a.K & 1) || (a.lda & 1) || (a.ldb & 1) || (a.strideA & 1) || (a.strideB & 1) || a.accumulate || a.ksplit != 1 ||
        (a.symmetric && a.N != 2 * a.M))
        return cudaErrorInvalidValue;
    const size_t smem = (size_t)V3_STAGES * (V3_BM + V3_BN) * V3_LD * sizeof(double);
    cudaError_t e = func_config(c, (const void*)k_vgemm3m, 128, smem, nullptr);
    if (e != cudaSuccess) return e;
    dim3 grid((a.N / 2 + V3_BN - 1) / V3_BN, (a.M + V3_BM - 1) / V3_BM, a.batch);
    k_vgemm3m<<<grid, 128, smem, st>>>(a);
    return cudaGetLastError();
}

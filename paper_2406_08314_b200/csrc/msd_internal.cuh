// Internal declarations shared by the translation units of libmsd_b200.so.
// Not part of the C ABI (include/msd.h).  sm_100a only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <map>
#include <string>
#include <utility>
#include <vector>

#define MSD_WT 8            // walkers per tile: lanes of a warp = 4 determinants x 8 walkers
#define MSD_MAX_LEVEL 16    // per-spin excitation level limit
#define MSD_MAX_NOCC 64     // electrons per spin limit
#define MSD_CF_MAX 4        // closed-form (register) minors up to this level; above: in-smem Gauss-Jordan

typedef double2 cplx;

__host__ __device__ __forceinline__ cplx cmake(double r, double i) { return make_double2(r, i); }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cneg(cplx a) { return make_double2(-a.x, -a.y); }
__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
    return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ cplx cscale(double s, cplx a) { return make_double2(s * a.x, s * a.y); }
// acc + a*b
__device__ __forceinline__ cplx cfma(cplx a, cplx b, cplx acc) {
    acc.x = fma(a.x, b.x, acc.x); acc.x = fma(-a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y); acc.y = fma(a.y, b.x, acc.y);
    return acc;
}
// acc - a*b
__device__ __forceinline__ cplx cfms(cplx a, cplx b, cplx acc) {
    acc.x = fma(-a.x, b.x, acc.x); acc.x = fma(a.y, b.y, acc.x);
    acc.y = fma(-a.x, b.y, acc.y); acc.y = fma(-a.y, b.x, acc.y);
    return acc;
}
__device__ __forceinline__ double cabs2(cplx a) { return a.x * a.x + a.y * a.y; }
__device__ __forceinline__ cplx cinv(cplx a) {
    // Smith-free: fine for the magnitudes here (no over/underflow guard needed for |a|^2 in range)
    double d = 1.0 / cabs2(a);
    return make_double2(a.x * d, -a.y * d);
}
__device__ __forceinline__ cplx cdiv(cplx a, cplx b) { return cmul(a, cinv(b)); }
__device__ __forceinline__ void red_add(cplx* p, cplx v) {
    atomicAdd(&p->x, v.x);
    atomicAdd(&p->y, v.y);
}
// CI-matrix accumulators are PLANAR per pair index x: C[x][0][WT] real parts, C[x][1][WT] imaginary parts, so that the
// 8 walkers of a determinant hit 64 contiguous bytes per reduction (measured in round 1: 2x the L2 reduction rate of
// interleaved complex).  p points at the lane's walker inside the tile.
__device__ __forceinline__ void red_add_planar(double* p, int x, cplx v) {
    atomicAdd(p + x * (2 * MSD_WT), v.x);
    atomicAdd(p + x * (2 * MSD_WT) + MSD_WT, v.y);
}
__device__ __forceinline__ cplx load_planar(const double* p, int x) {
    return make_double2(p[x * (2 * MSD_WT)], p[x * (2 * MSD_WT) + MSD_WT]);
}

// cp.async (16-byte, L2-only) and the FP64 tensor-core tile D(8x8) += A(8x4) B(4x8)
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, int src_bytes)
{
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// ---------------------------------------------------------------------------------------------
// packed trial (device pointers live in the context; this POD is passed to kernels by value)
// ---------------------------------------------------------------------------------------------
struct SpinDev {
    int n;                 // electrons of this spin
    int n_o, n_v;          // active occupied / active virtual orbitals (reading A10)
    int n_r;               // n + n_v : rows of L_sub
    int P;                 // n_o * n_v pair indices  x = p_loc * n_o + h_loc
    const int* occ_ref;    // [n]
    const int* act_v;      // [n_v] orbital index of active virtual r'
    const int* pos_o;      // [n_o] position in occ_ref of active occupied h_loc
    const double* Lsub;    // [(n_chol+1)][n_r][N]; slice n_chol holds the same rows of h1
};

struct Bucket {            // one (k_alpha, k_beta) level pair: determinants [start, start+count) of the sorted list
    int ka, kb;
    int64_t start, count;
    int64_t tab_off;       // byte offset of the bucket's rows in the table
    int rs;                // row stride in bytes (multiple of 4): [hA(ka) pA(ka) hB(kb) pB(kb)] local indices, uint8
};

struct WorkItem {          // a chunk of one bucket, processed by one CTA per walker tile
    int bucket;
    int ka, kb, rs;
    int64_t det_begin;     // in the sorted list
    int det_count;
    int64_t tab_off;       // byte offset of the chunk's first row
    int64_t sched_off;     // pull items (k_dets_pull): first entry of the item's pull list
    int64_t pull_off;      // pull items: first of the item's G + 1 piece boundaries (uint16, relative to sched_off)
};

// Force-bias CI reduction by OWNER PULL (k_dets_pull, dets.cu): nothing is scattered, no atomics.  For every chunk of
// determinants of one closed-form bucket the setup builds the list of all adjugate entries of the chunk, sorted by the unified
// pair index x they land on (alpha: x, beta: P_alpha + x),
//   C^s[x] = sum_{(I, a, b): x_ab(I) = x} c~_I R_I^sbar A_I^s[b][a],
// and cuts it into G contiguous pieces of (nearly) equal length whose ends fall on changes of x: piece q belongs to lane group q
// (8 lanes = 8 walkers) of the CTA, so every x has exactly one owner.
//   pass A  thread = (determinant, walker): R^a, R^b and, for spins of level >= 3, the adjugate by the division-free closed
//           forms; leaves the scale factors c~ R^b, c~ R^a and the (unscaled) level >= 3 adjugates in shared memory;
//   pass B  lane group q walks its piece: an entry is either recomputed from the shared-memory g tile (level 1: the scale
//           itself; level 2: one element of g) or read from the staged adjugate; the running sum of an x-run stays in
//           registers and is added to the CTA's C tile once per run.
// List entry (two words), everything pass B needs as ready-made byte offsets so that its inner loop has no branch on the level:
//   w0 = (2 det_local + spin) [10 bits: offset / 128 of the scale factor] | sign << 10 | x << 11 (14 bits) | last-of-run << 25
//   w1 = byte offset (walker 0, from the start of dynamic shared memory) of the value the scale multiplies: the constant 1.0
//        (level 1), one element of the g tile (level 2: the surviving element of the 2x2 minor), or one element of the staged
//        adjugate (levels 3, 4; it carries its own sign).
// Shared memory: C tile | 256 B (1.0) | pool = scale factors [D][2][8] + staged adjugates [E'][D][8] | g tile.
// Chunk sizes follow the pool: 256 B of scale factors per determinant plus 128 B per staged adjugate element.
#define PULL_DMAX 432      // determinants per chunk (12-bit det_local)

struct Workspace {
    int64_t wc = 0;        // walker capacity of one chunk (multiple of MSD_WT)
    int64_t want = 0;      // padded n_w the layout was made for
    int level = 0;         // 1 overlap, 2 force bias/greens, 3 energy, 4 propagation step : which buffers exist
    char* base = nullptr;  // one cudaMalloc
    size_t bytes = 0;
    // views
    cplx* theta[2] = {nullptr, nullptr};      // [wc][N][n]
    double* thetaT[2] = {nullptr, nullptr};   // [wc][n][2][N]  rows (w,i,c), K = N contiguous
    cplx* det0 = nullptr;                     // [wc][2]
    double* kappa2 = nullptr;                 // [wc][2]  (||O0||_F ||O0^-1||_F)^2 per walker and spin (energy level only)
    cplx* g[2] = {nullptr, nullptr};          // [nt][P][WT]
    double* C[2] = {nullptr, nullptr};        // [nt][P][2][WT] planar re/im (zeroed every call)
    cplx* Wacc = nullptr;                     // [wc]             (zeroed)
    cplx* E2nd = nullptr;                     // [wc]             (zeroed)
    cplx* E1nd = nullptr;                     // [wc]             (zeroed)
    cplx* FH[2] = {nullptr, nullptr};         // [nt][P][2][WT]   Hrot / F with the walker fastest (energy)
    int* wflags = nullptr;                    // [wc]
    double* Gp[2] = {nullptr, nullptr};       // [wc][2][n_r*N]   planar rows (w,c)
    cplx* Lam[2] = {nullptr, nullptr};        // [(n_chol+1)*n_r][wc][n]
    cplx* Bp[2] = {nullptr, nullptr};         // [wc][P][n_chol]
    cplx* Vab = nullptr;                      // [nt][Pa][Pb][WT]
    cplx* Vss[2] = {nullptr, nullptr};        // [nt][P][P][WT]
    cplx* F[2] = {nullptr, nullptr};          // [wc][P]          (zeroed)
    cplx* Hrot[2] = {nullptr, nullptr};       // [wc][P]
    cplx* Eacc = nullptr;                     // [wc][2]: (E1_0, E2_0)  (zeroed)
    cplx* X0 = nullptr;                       // [2][nw][n_chol] tr T^g per spin (zeroed)
    // propagation step (level 4 = force-bias buffers + these)
    cplx* fbuf = nullptr;                     // [wc][n_chol] force bias v
    double* Yf = nullptr;                     // [2 wc][ldg] shifted fields as the GEMM operand
    cplx* Aw = nullptr;                       // [wc][N][N] field matrices i sqrt(dt) sum_g y_g L^g
    cplx* ov_old = nullptr; cplx* ov_new = nullptr; cplx* expo = nullptr;     // [wc]
    int* fl_old = nullptr;                    // [wc]
    char* zero_begin = nullptr;               // region memset to 0 at the start of every chunk
    size_t zero_bytes = 0;
};

struct msd_ctx {
    int device = 0;
    int N = 0, n_chol = 0;
    int64_t n_det = 0;
    double e0 = 0.0;
    int n_sm = 148;
    struct SpinHost {
        int n = 0, n_o = 0, n_v = 0, n_r = 0, P = 0, kmax = 0;
        std::vector<int> occ_ref, act_o, act_v, pos_o;
        int* d_occ_ref = nullptr; int* d_act_v = nullptr; int* d_pos_o = nullptr;
        double* d_Lsub = nullptr;
    } sp[2];
    // packed determinant list
    unsigned char* d_tab = nullptr;
    double* d_coef = nullptr;
    std::vector<Bucket> buckets;
    std::vector<WorkItem> items_cf, items_gen, items_pull;
    WorkItem* d_items_cf = nullptr; WorkItem* d_items_gen = nullptr; WorkItem* d_items_pull = nullptr;
    unsigned short* d_pull_off = nullptr;     // per pull item: G + 1 piece boundaries
    uint2* d_pull_ent = nullptr;              // pull-list entries (see PULL_* above)
    int pull_class_begin[3] = {0, 0, 0};      // items_pull sorted by class: larger level <= 3 (512 threads), == 4 (256 threads)
    bool pull_gs = true;                      // the g tile sits in shared memory too
    size_t pull_pool = 0;                     // bytes of shared memory for scale factors + staged adjugates (0: pull disabled)
    int cf_class_begin[4] = {0, 0, 0, 0};      // items_cf is sorted by register class (larger level <=2, 3, 4)
    std::vector<int> gen_group_begin;         // items_gen is sorted by shared-memory group
    std::vector<int> gen_group_elems;         // ka^2+kb^2 bound of each group (complex elements per thread)
    // host copies for introspection
    std::vector<int64_t> h_perm; std::vector<double> h_coef; std::vector<int> h_ka, h_kb;
    Workspace ws;
    // device staging of the *_host entry points
    void* stg_a = nullptr; void* stg_b = nullptr; void* stg_out = nullptr; void* stg_flags = nullptr;
    size_t stg_a_bytes = 0, stg_b_bytes = 0, stg_out_bytes = 0, stg_flags_bytes = 0;
    int64_t ws_limit = 0;
    int64_t ws_limit_auto = 0;
    int64_t launches = 0;
    int no_smem_tiles = 0;                    // msd_set_option(MSD_OPT_NO_SMEM_TILES): test hook, see include/msd.h
    // propagation step (msd_propagator_setup / msd_propagate)
    double* d_LT = nullptr;                   // [N*N][ldg]  L with the Cholesky index contiguous
    double* d_hp = nullptr;                   // [N][ld]  h' of Eq. 4
    double* d_E = nullptr;                    // 3 x [ld][ld]: exp(-dt h'/2), the scaled matrix, scratch
    double prop_dt = 0.0; int prop_taylor = 0;
    const double* prop_x = nullptr; double* prop_w = nullptr;      // arguments of the running msd_propagate call
    cplx* fb_ovlp = nullptr;                  // msd_force_bias_overlap: where the running force-bias call also leaves the overlaps
    int shard_rank = 0, shard_world = 1;      // determinant sharding (msd_setup_sharded)
    void (*allreduce)(void*, void*, int64_t, void*) = nullptr; void* allreduce_user = nullptr;     // msd_set_allreduce
    int coop_min_elems = 50;                  // MSD_OPT_COOP_MIN_ELEMS: groups with ka^2+kb^2 above this run k_dets_coop, the rest k_dets_gen
    int coop_min_elems_fb = 72;               //   the same for the overlap / force-bias modes (measured crossovers: profiles/r02_sweep.md)
    bool noalloc_ready = false;               // msd_noalloc_setup ran on this context (msd_api.cu, no-allocation overlap call)
    double v3m_max_cond = 300.0;              // MSD_OPT_3M_MAX_COND: walkers whose reference block has ||O0||_F ||O0^-1||_F above this take the
                                              //   4-multiplication V contraction (accuracy: DESIGN.md section 7)
    bool no_3m = false;                       // MSD_OPT_NO_3M: V contractions by the 4-multiplication real form (test hook)
    bool no_fused = false;                    // MSD_OPT_NO_FUSED_S7: take the Lambda GEMM + dense kernel pair (test hook)
    bool need_lam = true;                     // the workspace holds the Lambda buffer (two-kernel S7 path)
    bool energy_ok = true;                    // the energy calls are supported for this trial (window size, see msd_setup)
    std::string energy_why;
    // launch configurations are fixed by the trial: occupancy per (kernel, block size, dynamic shared memory) is queried
    // once and kept here (func_config below), so the hot calls make no CUDA API call besides the launches themselves
    std::map<std::pair<const void*, size_t>, int> occ_cache;
    bool profiling = false;
    cudaEvent_t ev[8] = {};
    float phase_ms[6] = {};
    // fork/join side streams: independent launches of one call (the dets kernels of different register / shared-memory
    // classes, the per-spin GEMMs) run concurrently and rejoin the caller's stream before the call returns
    static constexpr int NAUX = 4;
    cudaStream_t aux[NAUX] = {};
    cudaEvent_t ev_fork = nullptr, ev_join[NAUX] = {};
    cudaEvent_t ev_done = nullptr;            // end of the most recent hot call (the workspace is free again after it)
    cudaStream_t last_stream = nullptr; bool have_done = false;
    std::string err;
    SpinDev dev(int s) const {
        SpinDev d; d.n = sp[s].n; d.n_o = sp[s].n_o; d.n_v = sp[s].n_v; d.n_r = sp[s].n_r; d.P = sp[s].P;
        d.occ_ref = sp[s].d_occ_ref; d.act_v = sp[s].d_act_v; d.pos_o = sp[s].d_pos_o; d.Lsub = sp[s].d_Lsub;
        return d;
    }
};

// ---------------------------------------------------------------------------------------------
// launchers (each returns cudaGetLastError() after its launches and bumps *launches)
// ---------------------------------------------------------------------------------------------
// pack.cu
cudaError_t launch_pack_mark(int64_t n_det, const int64_t* off, const int32_t* holes, const int32_t* parts, int N,
                             const int* pos_in_ref, int* used_h, int* used_p, int* err, cudaStream_t st);
cudaError_t launch_pack_rows(int64_t n_det, int N,
                             const int64_t* off_a, const int32_t* holes_a, const int32_t* parts_a,
                             const int64_t* off_b, const int32_t* holes_b, const int32_t* parts_b,
                             const int* occ_ref_a, int na, const int* occ_ref_b, int nb,
                             const int* pos_in_ref_a, const int* pos_in_ref_b,
                             const int* map_h_a, const int* map_p_a, const int* map_h_b, const int* map_p_b,
                             const double* ci, unsigned char* tmp_rows /*[n_det][64]*/, int* key, double* coef,
                             int* hist /*[17*17]*/, int* err, cudaStream_t st);
cudaError_t launch_pack_dedup(int64_t n_det, const unsigned char* tmp_rows, const int* key, int* slots, int64_t nslots,
                              int* err, cudaStream_t st);
cudaError_t launch_pack_scatter(int64_t n_det, const int* key, int n_buckets, const int* bucket_keys,
                                const int64_t* bucket_start, int64_t* perm, cudaStream_t st);
cudaError_t launch_pack_write(int64_t n_det, const int64_t* perm, const int* key, const unsigned char* tmp_rows,
                              const double* coef, int n_buckets, const Bucket* buckets, const int* bucket_of_key,
                              unsigned char* tab, double* coef_sorted, cudaStream_t st);
cudaError_t launch_pack_lsub(const double* L_or_h1, int n_slices, int N, int n_r, const int* rows,
                             double* out, cudaStream_t st);

// reference.cu
cudaError_t launch_reference(msd_ctx* c, int N, int ldN, SpinDev sa, SpinDev sb, int64_t nw,
                             const cplx* phi_a, const cplx* phi_b, Workspace& ws, bool want_thetaT, cudaStream_t st);

// dets.cu   mode: 0 overlap, 1 + CI matrix, 2 + second-order energy
cudaError_t launch_dets(msd_ctx* c, int mode, int64_t nw, Workspace& ws, cudaStream_t st);

// dense.cu
cudaError_t launch_green_rows(msd_ctx* c, int64_t nw, Workspace& ws, cplx* Gfull /*or null*/, cudaStream_t st);
cudaError_t launch_energy_dense(msd_ctx* c, int64_t nw, Workspace& ws, cudaStream_t st);
cudaError_t launch_energy_fused(msd_ctx* c, int64_t nw, Workspace& ws, cudaStream_t st);   // cudaErrorNotSupported: use the two-kernel path
bool energy_fused_shape(const msd_ctx* c, int* mtc, int* ntc, int* mtg, int* ntg, int* koff, int* Kv);
size_t energy_dense_smem(const msd_ctx* c, int GC);      // shared memory of the scalar S7 kernel with GC slices per CTA
cudaError_t launch_fx(msd_ctx* c, int64_t nw, Workspace& ws, cudaStream_t st);
cudaError_t launch_finish_overlap(msd_ctx* c, int64_t nw, Workspace& ws, cplx* ovlp, int* flags, cudaStream_t st);
cudaError_t launch_finish_energy(msd_ctx* c, int64_t nw, Workspace& ws, cplx* e, int64_t estride, int* flags, cudaStream_t st);
cudaError_t launch_fb_from_cb(msd_ctx* c, int64_t nw, Workspace& ws, cplx* out, int64_t ostride, cudaStream_t st);
cudaError_t launch_finish_flags(msd_ctx* c, int64_t nw, Workspace& ws, cplx* out, int64_t per_walker, int* flags,
                                cudaStream_t st);

// msd_api.cu : fork/join helper.  Fork f(c, st): launch i of a group goes to stream(i); join() makes st wait for all.
struct Fork {
    msd_ctx* c; cudaStream_t st; int used = 0; bool forked = false; cudaError_t err = cudaSuccess;
    Fork(msd_ctx* c_, cudaStream_t st_) : c(c_), st(st_) {}
    cudaStream_t stream(int i);     // i == 0: the caller's stream; i > 0: a side stream that waits for the fork point
    cudaError_t join();
};

// propagate.cu
cudaError_t prop_setup(msd_ctx* c, double dt, int n_taylor, const double* h1, const double* L, cudaStream_t st);
cudaError_t launch_prop_fields(msd_ctx* c, int64_t nw, const double* x, const cplx* v, double* Y, cplx* expo, cudaStream_t st);
cudaError_t launch_prop_vhs(msd_ctx* c, int64_t nw, const double* Y, cplx* Aw, cudaStream_t st);
cudaError_t launch_prop_orbitals(msd_ctx* c, int64_t nw, const cplx* Aw, cplx* phi_a, cplx* phi_b, cudaStream_t st);
cudaError_t launch_prop_finish(msd_ctx* c, int64_t nw, const cplx* ov_old, const cplx* ov_new, const cplx* expo, double* weights,
                               double* out, const int* fl_old, int* flags, cudaStream_t st);

// msd_api.cu : opt in to `smem` bytes of dynamic shared memory for `func` on the context's device (raised, never lowered,
// process-wide per device) and return the resident CTAs per SM for (nthr, smem); cached per context.
cudaError_t func_config(msd_ctx* c, const void* func, int nthr, size_t smem, int* occ);

// gemm.cu : C[m][n] (+)= sum_k A[m][k] * B[n][k]   (both K-contiguous, FP64 DMMA m8n8k4)
struct GemmArgs {
    const double* A; const double* B; double* C;
    int M, N, K;
    int64_t lda, ldb;           // row strides (doubles)
    int64_t strideA, strideB;   // per-batch strides (doubles); 0 = shared operand
    int batch;
    // output addressing: column pair (2j, 2j+1) of row m is one complex at
    //   C + 2*( (z / zdiv)*strideC_hi + (z % zdiv)*strideC_lo + m*cs_m + j*cs_j )   [complex units inside]
    int zdiv; int64_t strideC_hi, strideC_lo, cs_m, cs_j;
    int accumulate;             // 0: C = result; 1: C += result (plain read-modify-write); 2: RED.ADD (split-K)
    int ksplit = 1;             // grid.z = batch * ksplit; slice z % ksplit covers a BK-aligned K range (accumulate == 2)
    int bexpand = 0;            // 1: B holds N/2 COMPLEX rows (re,im interleaved along K); the kernel reads them as the real
                                //    rows (b_r, -b_i), (b_i, b_r) of a complex product, so that form is never written out
    // per-batch selection (V contractions): run batch z only if (max(sel[2z], sel[2z+1]) > sel_thr) == (sel_hi != 0);
    // a NaN counts as above the threshold
    const double* sel = nullptr; double sel_thr = 0.0; int sel_hi = 0;
    int symmetric = 0;          // 1: C is complex symmetric (M == N/2, A and B describe the same rows): only tiles that
                                //    touch the upper triangle are computed, element (m, j >= m) is also written to (j, m)
};
cudaError_t launch_gemm_tn(msd_ctx* c, const GemmArgs& a, cudaStream_t st);
cudaError_t launch_vgemm3m(msd_ctx* c, const GemmArgs& a, cudaStream_t st);     // complex bilinear product, 3-multiplication scheme

/* msd.h -- C ABI of the B200-native MSD-AFQMC Wick's-theorem hot path.
 *
 * Paper: "GPU-accelerated Auxiliary-field quantum Monte Carlo with multi-Slater determinant
 * trial states", arXiv 2406.08314 (text at /root/reference/PAPER.md; cited below as PAPER.md:L<line>).
 *
 * For a batch of walkers (single Slater determinants) against a multi-Slater-determinant
 * trial |Psi_T> = sum_I c_I |D_I> (Eq. 15; orthogonal CI expansion only) the library
 * evaluates, by the generalized Wick's theorem:
 *     the overlap <Psi_T|psi_w>                                              (Eq. 13 + Eq. 15)
 *     the mixed Green's function G^s_pq = <Psi_T|a+_p a_q|psi_w>/<Psi_T|psi_w>   (Eq. 14 generalised)
 *     the force bias v_g = sum_s sum_pq L^g_pq G^s_pq                            (Eq. 7 without -sqrt(dtau))
 *     the local (mixed) energy E = e0 + <Psi_T|H|psi_w>/<Psi_T|psi_w>, H of Eq. 2 with
 *         (pq|rs) = sum_g L^g_pq L^g_rs.
 *
 * Conventions:
 *   - a determinant is the ASCENDING-ordered string of its occupied orbitals, alpha string first;
 *     <D_I|psi> = det psi_a[occ_I^a,:] * det psi_b[occ_I^b,:].  The caller never supplies phases: the
 *     library computes the in-place -> sorted permutation parity itself.
 *   - G[p][q] = <a+_p a_q> = [phi (Psi_T^+ phi)^-1 Psi_T^+]_{qp}.
 *   - h1 is Eq. 2's h (NOT Eq. 3-4's h'); the two-body term is normal ordered.
 *   - CI coefficients are real.
 *
 * All arithmetic is float64 / complex128.  A complex128 is two consecutive doubles (re, im), i.e. the
 * memory of a contiguous torch.complex128 / numpy.complex128 array.
 *
 * Pointers marked HOST are read during the call and may be freed afterwards; pointers marked DEVICE must
 * be CUDA device memory on the context's device and stay valid until the work enqueued on `stream`
 * has completed.  `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 * The three hot calls enqueue kernels on `stream` and return without synchronising the host (the first
 * call for a larger n_w than seen before allocates workspace with cudaMalloc, which synchronises).
 * A context owns ONE workspace and one set of side streams: all calls on a context must be issued from one
 * host thread and are serialised against each other on the device (a call on another stream than the previous
 * call's first waits for that call's last kernel); use one context per concurrent stream.
 *
 * Errors: every function returning int returns MSD_OK (0) or a negative code; no exceptions cross the
 * ABI.  msd_last_error() gives a human-readable message for the last failure on that context (or the
 * last msd_setup failure if ctx is NULL).  Data-dependent singularities are NOT errors: a walker whose
 * reference overlap matrix is exactly singular (det O0 = 0) or whose W = sum_I c~_I R_I^a R_I^b is exactly
 * zero gets flags[w] != 0 (MSD_FLAG_*) and NaN outputs; the call still returns MSD_OK.
 */
#ifndef MSD_H
#define MSD_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MSD_OK            0
#define MSD_EINVAL       -1   /* bad argument or invalid excitation table */
#define MSD_ENOMEM       -2   /* host or device allocation failed */
#define MSD_ECUDA        -3   /* a CUDA runtime call or kernel launch failed */
#define MSD_EUNSUPPORTED -4   /* size outside what the kernels support (see msd_setup) */

#define MSD_FLAG_SINGULAR_REFERENCE 1   /* det psi[occ_ref,:] == 0 for a spin */
#define MSD_FLAG_ZERO_OVERLAP       2   /* W == 0 */

typedef struct msd_ctx msd_ctx;   /* opaque; owns every device copy made at setup and all workspace */

/* msd_setup: build the trial (PAPER.md:L222-254 inputs h1e, chol, e0, (coeff, occa, occb) in
 * hole/particle form; S0 "pack" of SURVEY.md 8(a)).  Runs the excitation-table packer kernels
 * (validate, phases, level sort into contiguous buckets) and packs the rows of L and h1 that the path touches.
 *   N, n_alpha, n_beta, n_chol, n_det : sizes.  Limits, ALL checked here (else MSD_EUNSUPPORTED): 1 <= N <= 1024,
 *       0 <= n_s <= 64, n_s <= N, n_chol >= 1, 1 <= n_det < 2^31, per-spin excitation level <= 16 and
 *       k_alpha^2 + k_beta^2 <= 400 for every determinant, active window per spin (n_o distinct hole orbitals,
 *       n_v distinct particle orbitals) n_o, n_v <= 255 and n_o*n_v <= 8192.
 *       The energy calls (msd_local_energy, msd_force_bias_energy) additionally need n_o*n_v <= 4096 per spin
 *       (they hold (n_o n_v)^2 two-body tensors per walker) and, for windows wider than 16 x 16, that
 *       n^2 + 2 n n_v + 2 n_o n_v complex numbers per spin fit in 227 KB of shared memory: a wider trial still sets
 *       up -- overlap, force bias and Green's function work -- msd_get_info()[8] is 0 and the energy calls return
 *       MSD_EUNSUPPORTED.
 *   h1   HOST [N][N] row-major, real symmetric.
 *   L    HOST [n_chol][N][N], each slice real symmetric.
 *   e0   constant added to every energy.
 *   occ_ref_a/b  HOST [n_alpha]/[n_beta], strictly ascending reference occupation.
 *   exc_off_s HOST [n_det+1] CSR offsets; determinant I has level k = off[I+1]-off[I] in spin s;
 *   holes_s / parts_s HOST [off[n_det]]: holes are in occ_ref_s, particles are not; distinct within a
 *       determinant; any order (the a-th smallest hole is paired with the a-th smallest particle).
 *   ci   HOST [n_det] real coefficients in the ascending-string convention.
 *   stream: setup work is enqueued there and synchronised before returning.
 * On success *out is a new context (destroy with msd_destroy).  Invalid tables -> MSD_EINVAL: an index out of
 * range, a hole outside / a particle inside the reference, an orbital repeated inside a determinant, a level
 * above n_s, or the same determinant listed twice (the CI expansion is orthogonal, Eq. 15). */
int msd_setup(msd_ctx** out, int N, int n_alpha, int n_beta, int n_chol, int64_t n_det,
              const double* h1, const double* L, double e0,
              const int32_t* occ_ref_a, const int32_t* occ_ref_b,
              const int64_t* exc_off_a, const int32_t* holes_a, const int32_t* parts_a,
              const int64_t* exc_off_b, const int32_t* holes_b, const int32_t* parts_b,
              const double* ci, void* stream);

/* Determinant-sharded multi-GPU (the paper's stated next step).
 * msd_setup_sharded builds the same trial, but the context evaluates only slice shard_rank of shard_world of every level
 * bucket of the determinant list (every rank passes the WHOLE trial: active window, table order and introspection are those of
 * the whole trial; msd_setup = shard 0 of 1).  A hot call on a sharded context needs the partial sums of all ranks:
 * msd_set_allreduce registers a hook that the call invokes, on the host, once after each determinant pass with
 *     buf        DEVICE float64 [n]: this rank's partial C^alpha, C^beta, W, E2nd, E1nd of the walker chunk (one contiguous run),
 *     stream     the stream the call is enqueued on (the library has synchronised it: the partial sums are complete);
 * the hook must perform, or enqueue on `stream`, an in-place SUM of buf over the ranks (e.g. ncclAllReduce / torch.distributed.all_reduce;
 * n is about (2 + 2 n_o n_v) complex per walker: 0.7 MB at 100 walkers of a 15 x 15 window) and return.  Every rank must make the
 * same calls with the same walkers.  Everything that is not a sum over determinants (reference step, dense contractions) is
 * replicated on every rank.  fn == NULL removes the hook. */
typedef void (*msd_allreduce_fn)(void* user, void* buf, int64_t n, void* stream);
int msd_setup_sharded(msd_ctx** out, int N, int n_alpha, int n_beta, int n_chol, int64_t n_det,
                      const double* h1, const double* L, double e0,
                      const int32_t* occ_ref_a, const int32_t* occ_ref_b,
                      const int64_t* exc_off_a, const int32_t* holes_a, const int32_t* parts_a,
                      const int64_t* exc_off_b, const int32_t* holes_b, const int32_t* parts_b,
                      const double* ci, int shard_rank, int shard_world, void* stream);
int msd_set_allreduce(msd_ctx* ctx, msd_allreduce_fn fn, void* user);

/* Convenience for the paper's (coeff, occa, occb) format: occa HOST [n_det][n_alpha],
 * occb HOST [n_det][n_beta] occupation lists (any order inside a row); determinant 0 is the reference. */
int msd_setup_from_occ(msd_ctx** out, int N, int n_alpha, int n_beta, int n_chol, int64_t n_det,
                       const double* h1, const double* L, double e0,
                       const int32_t* occa, const int32_t* occb, const double* ci, void* stream);

/* Walkers: phi_a DEVICE [n_w][N][n_alpha] complex128 row-major, phi_b DEVICE [n_w][N][n_beta]; columns need
 * not be orthonormal.  flags DEVICE [n_w] int32 or NULL.  n_w >= 0 (0 is a no-op). */

/* ovlp DEVICE [n_w] complex128 = <Psi_T|psi_w>  (S1, S2, S4 of SURVEY.md 8(a)). */
int msd_overlap(msd_ctx* ctx, int64_t n_w, const void* phi_a, const void* phi_b,
                void* ovlp, int32_t* flags, void* stream);

/* fb DEVICE [n_w][n_chol] complex128 = sum_s sum_pq L^g_pq G^s_pq[w]   (Eq. 7 without -sqrt(dtau); the caller
 * scales: reading A4).  S1-S6. */
int msd_force_bias(msd_ctx* ctx, int64_t n_w, const void* phi_a, const void* phi_b,
                   void* fb, int32_t* flags, void* stream);

/* Conditioning of the walkers' reference blocks O0 = psi[occ_ref, :]: cond DEVICE [n_w][2] float64 =
 * ||O0||_F ||O0^-1||_F per walker and spin (about 2-4 x the 2-norm condition number; inf for a singular block, 0 for a spin
 * without electrons).  This is the quantity the accuracy of msd_local_energy depends on (see there): walkers beyond
 * ~2000 carry energy errors above 1e-8 Ha (1e-5 Ha measured at 1e4) and are better re-orthonormalised or evaluated otherwise. */
int msd_reference_cond(msd_ctx* ctx, int64_t n_w, const void* phi_a, const void* phi_b, double* cond, void* stream);

/* msd_force_bias with the overlaps of the same walkers from the same determinant pass (the pass forms W = sum_I c_I R_I
 * and det O0 anyway; a propagation step needs both: PAPER.md Eq. 7 and Eq. 8): fb as in msd_force_bias, ovlp DEVICE [n_w]
 * as in msd_overlap.  Saves the separate msd_overlap call (0.5 ms of 2.7 ms at the Fe2S2-shaped config). */
int msd_force_bias_overlap(msd_ctx* ctx, int64_t n_w, const void* phi_a, const void* phi_b,
                           void* fb, void* ovlp, int32_t* flags, void* stream);

/* e DEVICE [n_w][3] complex128 = (E, E1, E2): E = e0 + E1 + E2, E1 one-body, E2 two-body.  S1-S9.
 * Accuracy: everything is expressed through Theta = psi (psi[occ_ref,:])^-1 (Wick's theorem around the reference
 * determinant), so the FP64 error of the energies grows with the conditioning of the walker's reference block O0 =
 * psi[occ_ref,:]: about 3e-13 Ha at cond_2(O0) ~ 30, 3e-10 at 200, 4e-9 at 700-900, and beyond 1e-8 Ha (5e-8 measured at
 * cond_2 = 938) for worse walkers; overlaps and force bias stay within relative 2e-11 there.  A
 * population whose walkers are re-orthonormalised regularly stays far below these values. */
int msd_local_energy(msd_ctx* ctx, int64_t n_w, const void* phi_a, const void* phi_b,
                     void* e, int32_t* flags, void* stream);

/* Force bias AND local energy of the same walkers in one pass (the metric's unit of work: one force-bias + local-energy
 * evaluation per walker x determinant).  out DEVICE [n_w][n_chol + 3] complex128: out[w][0..n_chol) = fb as in
 * msd_force_bias, out[w][n_chol..n_chol+3) = (E, E1, E2) as in msd_local_energy.  The determinant kernels run once:
 * the energy pass also accumulates the CI matrix C, and the force bias is taken from C and the half-rotated Cholesky
 * slices B^g that the energy path holds,  fb_g = sum_s [ X0^s_g + (1/W) sum_x C^s[x] B^{s,g}[x] ]  -- the same
 * quantity as Eq. 7 / msd_force_bias, not a different estimator.  S1-S9. */
int msd_force_bias_energy(msd_ctx* ctx, int64_t n_w, const void* phi_a, const void* phi_b,
                          void* out, int32_t* flags, void* stream);

/* G DEVICE [n_w][2][N][N] complex128, G[w][s][p][q] = <a+_p a_q>.  Test hook (S5). */
int msd_greens(msd_ctx* ctx, int64_t n_w, const void* phi_a, const void* phi_b,
               void* G, int32_t* flags, void* stream);

/* One phaseless-AFQMC propagation step around the hot path (Eq. 5, Eq. 7-12).
 *
 * msd_propagator_setup fixes the time step dt > 0 and the order n_taylor (1..64) of the Taylor series that applies the field
 * exponential, builds h' = h - 1/2 sum_g L^g L^g (Eq. 4) and exp(-dt h'/2) on the device (scaling and squaring), and keeps L
 * with the Cholesky index contiguous (N^2 x n_chol doubles of device memory).  h1, L: the HOST arrays msd_setup was given.
 * May be called again to change dt.  Synchronises `stream`.
 *
 * msd_propagate advances every walker of the batch by one step, IN PLACE:
 *     v = force bias (as msd_force_bias),  xbar = -i sqrt(dt) v                              Eq. 7 (reading A20)
 *     psi <- B(x - xbar) psi,  B(y) = exp(-dt h'/2) exp(i sqrt(dt) sum_g y_g L^g) exp(-dt h'/2)     Eq. 5
 *     S = <Psi_T|psi_new>/<Psi_T|psi_old>,  theta = arg S                                    Eq. 8-9
 *     I = S exp(x.xbar - xbar.xbar/2),  I_ph = |I| max(0, cos theta),  w <- I_ph w           Eq. 10-12
 *   phi_a, phi_b  DEVICE walkers as above, overwritten with the propagated (not re-orthonormalised) walkers.
 *   x        DEVICE [n_w][n_chol] float64: the auxiliary fields, drawn by the caller (standard normal).
 *   weights  DEVICE [n_w] float64, multiplied by I_ph in place; may be NULL.
 *   step_out DEVICE [n_w][8] float64: (Re S, Im S, theta, I_ph, Re <Psi_T|psi_new>, Im <Psi_T|psi_new>, Re I, Im I).
 *   flags    DEVICE [n_w] or NULL: MSD_FLAG_* of the old OR the new walker (NaN outputs for those).
 * Population control and re-orthogonalisation are the caller's. */
int msd_propagator_setup(msd_ctx* ctx, double dt, int n_taylor, const double* h1, const double* L, void* stream);
int msd_propagate(msd_ctx* ctx, int64_t n_w, void* phi_a, void* phi_b, const double* x, double* weights,
                  double* step_out, int32_t* flags, void* stream);

/* HOST-buffer variants of the hot calls (the end-to-end path: bench.py's "e2e").  phi_a / phi_b / the result /
 * flags are HOST pointers with the same layouts as above (pinned memory makes the copies asynchronous, pageable
 * memory works too).  Each call enqueues on `stream`: host->device copy of the walkers into staging buffers owned by
 * the context, the same kernels as the device variant, device->host copy of the result (and flags); it then
 * synchronises `stream`, so the result is valid on return.  Same return codes. */
int msd_overlap_host(msd_ctx* ctx, int64_t n_w, const void* phi_a, const void* phi_b,
                     void* ovlp, int32_t* flags, void* stream);
int msd_force_bias_host(msd_ctx* ctx, int64_t n_w, const void* phi_a, const void* phi_b,
                        void* fb, int32_t* flags, void* stream);
int msd_local_energy_host(msd_ctx* ctx, int64_t n_w, const void* phi_a, const void* phi_b,
                          void* e, int32_t* flags, void* stream);
int msd_force_bias_energy_host(msd_ctx* ctx, int64_t n_w, const void* phi_a, const void* phi_b,
                               void* out, int32_t* flags, void* stream);

/* Introspection of the packed trial (host-side copies made at setup; for tests of the packer).
 * msd_get_info fills info[0..10]: [0]=n_o_alpha, [1]=n_v_alpha, [2]=n_o_beta, [3]=n_v_beta, [4]=number of level
 * buckets, [5]=max level alpha, [6]=max level beta, [7]=walker tile width, [8]=1 if the energy calls are supported,
 * [9]=shard rank, [10]=shard count.
 * msd_get_packed copies, in the packer's sorted order, perm[n_det] (original index of each packed
 * determinant), coef[n_det] (c_I * phase_a * phase_b), level_a[n_det], level_b[n_det]; any may be NULL. HOST. */
int msd_get_info(const msd_ctx* ctx, int64_t* info11);
int msd_get_packed(const msd_ctx* ctx, int64_t* perm, double* coef, int32_t* level_a, int32_t* level_b);

/* Set an upper bound (bytes) on the workspace the hot calls may allocate (default: 70 % of free device
 * memory at the first call); walkers are processed in chunks that fit. */
int msd_set_workspace_limit(msd_ctx* ctx, int64_t bytes);

/* No-allocation variant of msd_overlap, for callers that cannot allocate in the hot loop (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc).  Same arguments, same result as msd_overlap (same kernels; sums
 * in the same order up to the order of atomic adds), but the call's workspace -- zeroed per-walker accumulators, Theta, g,
 * det0 of the walkers -- lives in ONE file-scope device array of MSD_NOALLOC_SCRATCH_BYTES inside the library instead of
 * the context's cudaMalloc'ed workspace; every GPU that loads the library holds that array until the process exits.
 *   msd_noalloc_setup(ctx, stream): SET-UP, once per context, with the context's device current, outside the
 *       no-allocation region: resolves the array's device address for this device and creates the context's side streams
 *       and events (this call MAY allocate).  Determinant-sharded contexts: MSD_EUNSUPPORTED.
 *   msd_overlap_noalloc(...): calls no cudaMalloc / cudaFree / stream or event creation and no allocating library routine;
 *       it launches kernels and records / waits on the context's existing events only.  Without a prior msd_noalloc_setup
 *       on the context: MSD_EINVAL.  The whole batch must fit: n_w walkers need about
 *       16 B x ceil8(n_w) x (5 + sum_sigma (N n_sigma + 2 n_o n_v)) bytes (ceil8: rounded up to a multiple of 8; e.g. up to
 *       48 walkers of N = 100, n_alpha = n_beta = 20 with a
 *       15 x 15 active window); a larger batch is refused with MSD_ENOMEM and a message that states both sizes -- split the
 *       batch or use msd_overlap.  n_w = 0 is a no-op.
 *   The array is shared by every context and every call on the device and keeps the last call's contents; the accumulators
 *   are cleared at the start of each call.  Calls that overlap on the GPU (different streams, host threads or contexts)
 *   RACE on it: the caller keeps them ordered (one stream, or events).  It does not interfere with the other calls of the
 *   context, which keep their own workspace. */
#define MSD_NOALLOC_SCRATCH_BYTES (4 * 1024 * 1024)
int msd_noalloc_setup(msd_ctx* ctx, void* stream);
int msd_overlap_noalloc(msd_ctx* ctx, int64_t n_w, const void* phi_a, const void* phi_b,
                        void* ovlp, int32_t* flags, void* stream);

/* Number of kernels the library launched on this context since setup (for bench.py's gpu_launches). */
int64_t msd_launch_count(const msd_ctx* ctx);

/* Per-phase device timings of the most recent hot call when profiling is enabled with
 * msd_set_profiling(ctx, 1): fills ms[0..n-1] for phases (reference, dets, greens/fb, dense, vgemm, assemble);
 * synchronises the stream.  Off by default (no events recorded). */
int msd_set_profiling(msd_ctx* ctx, int on);
int msd_get_phase_ms(msd_ctx* ctx, float* ms, int n);

/* Options (arguments of the context, no environment variables are read).
 *   MSD_OPT_NO_SMEM_TILES (value 0, 1 or 2; default 0): TEST HOOK.  Forces the kernel variants that are otherwise chosen
 *       only for active windows too wide for shared memory, so that those paths can be parity-tested on small inputs:
 *       1 = a walker tile's CI matrix / Hrot / F do not fit (RED.ADD scatter of C, Hrot / F through L1);
 *       2 = the tile's g slices do not fit either (n_o n_v summed over spins above ~1600: g through L1 as well).
 *       Results are the same.  Unknown option or value: MSD_EINVAL.
 *   MSD_OPT_NO_FUSED_S7 (0 / 1; default 0): TEST HOOK.  1 takes the two-kernel form of the half rotation (Lambda = L_sub Theta
 *       written to memory by the GEMM, dense intermediates by a second kernel) that otherwise only runs for shapes the fused
 *       kernel does not cover.  Results are the same.
 *   MSD_OPT_NO_3M (0 / 1; default 0): TEST HOOK.  1 computes the V contractions with the four-multiplication real form of the
 *       complex product (k_gemm_tn) instead of the three-multiplication kernel (k_vgemm3m).  Same results to rounding.
 *   MSD_OPT_3M_MAX_COND (value >= 0; default 300): ACCURACY KNOB.  The V contractions of the energy calls use the
 *       3-multiplication complex product for the walkers whose reference block O0 = psi[occ_ref, :] has
 *       ||O0||_F ||O0^-1||_F <= value and the 4-multiplication product for the others (chosen per walker on the device; the
 *       3-multiplication form is 20 % faster but loses 4-15 x more digits on ill-conditioned walkers: DESIGN.md section 7).
 *       0 = the 4-multiplication product for every walker (same as MSD_OPT_NO_3M = 1); a huge value = always 3 multiplications.
 *   MSD_OPT_COOP_MIN_ELEMS (0..200; default 50 for the energy calls, 72 for overlap / force bias): TUNING KNOB / TEST HOOK.  Determinant buckets with an
 *       excitation level above 4 in either spin and ka^2 + kb^2 above this value run the warp-cooperative kernel (one
 *       determinant x 8 walkers per warp, 4 helper lanes per walker); the others keep one determinant per thread.  Same
 *       results to rounding (the two kernels sum the same terms in different orders). */
#define MSD_OPT_NO_SMEM_TILES 1
#define MSD_OPT_NO_FUSED_S7 2
#define MSD_OPT_NO_3M 3
#define MSD_OPT_COOP_MIN_ELEMS 4
#define MSD_OPT_3M_MAX_COND 5
int msd_set_option(msd_ctx* ctx, int option, int64_t value);

void msd_destroy(msd_ctx* ctx);
const char* msd_last_error(const msd_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* MSD_H */

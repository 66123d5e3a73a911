// S0 "pack": excitation-table packer kernels run once in msd_setup.
//   PAPER.md:L297 "each set handles single, double, triple, and n-fold excitation components" ->
//   determinants are sorted by per-spin excitation level pair (k_alpha, k_beta) into contiguous buckets;
//   reading A6/A7: the phase is the parity of the permutation that sorts the reference list
//   with h_a -> p_a substituted in place (a-th smallest hole paired with a-th smallest particle).
#include "msd_internal.cuh"

#define ERR_RANGE 1
#define ERR_HOLE_NOT_OCC 2
#define ERR_PART_IS_OCC 4
#define ERR_REPEATED 8
#define ERR_LEVEL 16
#define ERR_DUPLICATE 32

__global__ void k_pack_mark(int64_t n_det, const int64_t* __restrict__ off, const int32_t* __restrict__ holes,
                            const int32_t* __restrict__ parts, int N, const int* __restrict__ pos_in_ref,
                            int* used_h, int* used_p, int* err)
{
    int64_t I = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (I >= n_det) return;
    int64_t b = off[I], e = off[I + 1];
    if (e < b || e - b > MSD_MAX_LEVEL) { atomicOr(err, ERR_LEVEL); return; }
    for (int64_t t = b; t < e; t++) {
        int h = holes[t], p = parts[t];
        if (h < 0 || h >= N || p < 0 || p >= N) { atomicOr(err, ERR_RANGE); continue; }
        if (pos_in_ref[h] < 0) atomicOr(err, ERR_HOLE_NOT_OCC); else used_h[h] = 1;
        if (pos_in_ref[p] >= 0) atomicOr(err, ERR_PART_IS_OCC); else used_p[p] = 1;
    }
}

// sort ascending (insertion), return nonzero if a value repeats
__device__ int sort_small(int* a, int k)
{
    for (int i = 1; i < k; i++) {
        int v = a[i], j = i - 1;
        while (j >= 0 && a[j] > v) { a[j + 1] = a[j]; j--; }
        a[j + 1] = v;
    }
    int rep = 0;
    for (int i = 1; i < k; i++) rep |= (a[i] == a[i - 1]);
    return rep;
}

// parity (+1/-1) of the permutation that sorts occ_ref with holes[a] -> parts[a] substituted in place
__device__ double phase_inplace(const int* __restrict__ occ_ref, int n, const int* __restrict__ pos_in_ref,
                                const int* h, const int* p, int k)
{
    int lst[MSD_MAX_NOCC];
    for (int i = 0; i < n; i++) lst[i] = occ_ref[i];
    for (int a = 0; a < k; a++) lst[pos_in_ref[h[a]]] = p[a];
    int inv = 0;
    for (int i = 0; i < n; i++)
        for (int j = i + 1; j < n; j++) inv += (lst[i] > lst[j]);
    return (inv & 1) ? -1.0 : 1.0;
}

__global__ void k_pack_rows(int64_t n_det, int N,
                            const int64_t* __restrict__ off_a, const int32_t* __restrict__ holes_a,
                            const int32_t* __restrict__ parts_a,
                            const int64_t* __restrict__ off_b, const int32_t* __restrict__ holes_b,
                            const int32_t* __restrict__ parts_b,
                            const int* __restrict__ occ_ref_a, int na, const int* __restrict__ occ_ref_b, int nb,
                            const int* __restrict__ pos_a, const int* __restrict__ pos_b,
                            const int* __restrict__ map_h_a, const int* __restrict__ map_p_a,
                            const int* __restrict__ map_h_b, const int* __restrict__ map_p_b,
                            const double* __restrict__ ci, unsigned char* tmp_rows, int* key, double* coef,
                            int* hist, int* err)
{
    int64_t I = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (I >= n_det) return;
    unsigned char* row = tmp_rows + I * 64;
    double ph = 1.0;
    int kk[2];
    int o = 0;
    for (int s = 0; s < 2; s++) {
        const int64_t* off = s ? off_b : off_a;
        const int32_t* holes = s ? holes_b : holes_a;
        const int32_t* parts = s ? parts_b : parts_a;
        const int* occ_ref = s ? occ_ref_b : occ_ref_a;
        const int* pos = s ? pos_b : pos_a;
        const int* map_h = s ? map_h_b : map_h_a;
        const int* map_p = s ? map_p_b : map_p_a;
        int n = s ? nb : na;
        int k = (int)(off[I + 1] - off[I]);
        int h[MSD_MAX_LEVEL], p[MSD_MAX_LEVEL];
        for (int a = 0; a < k; a++) { h[a] = holes[off[I] + a]; p[a] = parts[off[I] + a]; }
        if (sort_small(h, k) | sort_small(p, k)) atomicOr(err, ERR_REPEATED);
        if (k > n) atomicOr(err, ERR_LEVEL);
        ph *= phase_inplace(occ_ref, n, pos, h, p, k);
        for (int a = 0; a < k; a++) row[o + a] = (unsigned char)map_h[h[a]];
        for (int a = 0; a < k; a++) row[o + k + a] = (unsigned char)map_p[p[a]];
        o += 2 * k;
        kk[s] = k;
    }
    int ky = kk[0] * (MSD_MAX_LEVEL + 1) + kk[1];
    key[I] = ky;
    coef[I] = ci[I] * ph;
    atomicAdd(&hist[ky], 1);
}

// Duplicate determinants (Eq. 15 is an orthogonal expansion: every determinant once).  Exact, not probabilistic: an
// open-addressing table of determinant indices keyed by a hash of (level key, packed row); a probe that meets an occupied
// slot compares the full rows and either reports the duplicate or moves on to the next slot.
__global__ void k_pack_dedup(int64_t n_det, const unsigned char* __restrict__ tmp_rows, const int* __restrict__ key,
                             int* slots, int64_t nslots, int* err)
{
    int64_t I = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (I >= n_det) return;
    const int ky = key[I];
    const int nb = 2 * (ky / (MSD_MAX_LEVEL + 1)) + 2 * (ky % (MSD_MAX_LEVEL + 1));
    const unsigned char* row = tmp_rows + I * 64;
    unsigned long long h = 1469598103934665603ull ^ (unsigned long long)ky;       // FNV-1a
    for (int t = 0; t < nb; t++) { h ^= row[t]; h *= 1099511628211ull; }
    h ^= h >> 29;
    int64_t s = (int64_t)(h & (unsigned long long)(nslots - 1));
    for (;;) {
        const int prev = atomicCAS(&slots[s], -1, (int)I);
        if (prev == -1) return;
        if (key[prev] == ky) {
            const unsigned char* other = tmp_rows + (int64_t)prev * 64;
            bool same = true;
            for (int t = 0; t < nb; t++) same &= (other[t] == row[t]);
            if (same) { atomicOr(err, ERR_DUPLICATE); return; }
        }
        s = (s + 1) & (nslots - 1);
    }
}

// stable counting-sort scatter: block b owns bucket b, walks the keys in order
__global__ void k_pack_scatter(int64_t n_det, const int* __restrict__ key, const int* __restrict__ bucket_keys,
                               const int64_t* __restrict__ bucket_start, int64_t* perm)
{
    const int mine = bucket_keys[blockIdx.x];
    int64_t base = bucket_start[blockIdx.x];
    __shared__ int warp_cnt[32];
    __shared__ int total;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    for (int64_t c0 = 0; c0 < n_det; c0 += blockDim.x) {
        int64_t I = c0 + threadIdx.x;
        bool f = (I < n_det) && (key[I] == mine);
        unsigned m = __ballot_sync(0xffffffffu, f);
        int before = __popc(m & ((1u << lane) - 1));
        if (lane == 0) warp_cnt[wid] = __popc(m);
        __syncthreads();
        if (threadIdx.x == 0) {
            int acc = 0;
            for (int w = 0; w < nwarp; w++) { int t = warp_cnt[w]; warp_cnt[w] = acc; acc += t; }
            total = acc;
        }
        __syncthreads();
        if (f) perm[base + warp_cnt[wid] + before] = I;
        base += total;
        __syncthreads();
    }
}

__global__ void k_pack_write(int64_t n_det, const int64_t* __restrict__ perm, const int* __restrict__ key,
                             const unsigned char* __restrict__ tmp_rows, const double* __restrict__ coef,
                             const Bucket* __restrict__ buckets, const int* __restrict__ bucket_of_key,
                             unsigned char* tab, double* coef_sorted)
{
    int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_det) return;
    int64_t I = perm[s];
    Bucket b = buckets[bucket_of_key[key[I]]];
    unsigned char* row = tab + b.tab_off + (s - b.start) * b.rs;
    const unsigned char* src = tmp_rows + I * 64;
    int nb = 2 * b.ka + 2 * b.kb;
    for (int t = 0; t < b.rs; t++) row[t] = (t < nb) ? src[t] : (unsigned char)0;
    coef_sorted[s] = coef[I];
}

// L_sub[slice][r][q] = L[slice][rows[r]][q]   (A17: rows of L the path touches)
__global__ void k_pack_lsub(const double* __restrict__ L, int N, int n_r, const int* __restrict__ rows,
                            double* __restrict__ out)
{
    int slice = blockIdx.y, r = blockIdx.x;
    const double* src = L + ((int64_t)slice * N + rows[r]) * N;
    double* dst = out + ((int64_t)slice * n_r + r) * N;
    for (int q = threadIdx.x; q < N; q += blockDim.x) dst[q] = src[q];
}

cudaError_t launch_pack_mark(int64_t n_det, const int64_t* off, const int32_t* holes, const int32_t* parts, int N,
                             const int* pos_in_ref, int* used_h, int* used_p, int* err, cudaStream_t st)
{
    int thr = 256;
    k_pack_mark<<<(unsigned)((n_det + thr - 1) / thr), thr, 0, st>>>(n_det, off, holes, parts, N, pos_in_ref,
                                                                    used_h, used_p, err);
    return cudaGetLastError();
}

cudaError_t launch_pack_rows(int64_t n_det, int N,
                             const int64_t* off_a, const int32_t* holes_a, const int32_t* parts_a,
                             const int64_t* off_b, const int32_t* holes_b, const int32_t* parts_b,
                             const int* occ_ref_a, int na, const int* occ_ref_b, int nb,
                             const int* pos_in_ref_a, const int* pos_in_ref_b,
                             const int* map_h_a, const int* map_p_a, const int* map_h_b, const int* map_p_b,
                             const double* ci, unsigned char* tmp_rows, int* key, double* coef,
                             int* hist, int* err, cudaStream_t st)
{
    int thr = 128;
    k_pack_rows<<<(unsigned)((n_det + thr - 1) / thr), thr, 0, st>>>(
        n_det, N, off_a, holes_a, parts_a, off_b, holes_b, parts_b, occ_ref_a, na, occ_ref_b, nb,
        pos_in_ref_a, pos_in_ref_b, map_h_a, map_p_a, map_h_b, map_p_b, ci, tmp_rows, key, coef, hist, err);
    return cudaGetLastError();
}

cudaError_t launch_pack_dedup(int64_t n_det, const unsigned char* tmp_rows, const int* key, int* slots, int64_t nslots,
                              int* err, cudaStream_t st)
{
    int thr = 256;
    k_pack_dedup<<<(unsigned)((n_det + thr - 1) / thr), thr, 0, st>>>(n_det, tmp_rows, key, slots, nslots, err);
    return cudaGetLastError();
}

cudaError_t launch_pack_scatter(int64_t n_det, const int* key, int n_buckets, const int* bucket_keys,
                                const int64_t* bucket_start, int64_t* perm, cudaStream_t st)
{
    k_pack_scatter<<<n_buckets, 1024, 0, st>>>(n_det, key, bucket_keys, bucket_start, perm);
    return cudaGetLastError();
}

cudaError_t launch_pack_write(int64_t n_det, const int64_t* perm, const int* key, const unsigned char* tmp_rows,
                              const double* coef, int n_buckets, const Bucket* buckets, const int* bucket_of_key,
                              unsigned char* tab, double* coef_sorted, cudaStream_t st)
{
    (void)n_buckets;
    int thr = 256;
    k_pack_write<<<(unsigned)((n_det + thr - 1) / thr), thr, 0, st>>>(n_det, perm, key, tmp_rows, coef, buckets,
                                                                     bucket_of_key, tab, coef_sorted);
    return cudaGetLastError();
}

cudaError_t launch_pack_lsub(const double* L, int n_slices, int N, int n_r, const int* rows, double* out,
                             cudaStream_t st)
{
    if (n_r == 0 || n_slices == 0) return cudaSuccess;
    dim3 grid(n_r, n_slices);
    k_pack_lsub<<<grid, 128, 0, st>>>(L, N, n_r, rows, out);
    return cudaGetLastError();
}

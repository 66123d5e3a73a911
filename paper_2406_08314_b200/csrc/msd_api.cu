// C ABI of libmsd_b200.so (include/msd.h): context, setup (S0), workspace, and the call graphs of the hot calls.
#include "../../include/msd.h"
#include "msd_internal.cuh"

#include <algorithm>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>

static std::string g_setup_error;

// cudaFuncAttributeMaxDynamicSharedMemorySize is state of the (device, function) pair shared by every context of the
// process: it is only ever raised, under a lock; occupancy is cached per context.
static std::mutex g_func_mutex;
static std::map<std::pair<int, const void*>, size_t> g_func_smem;

cudaError_t func_config(msd_ctx* c, const void* func, int nthr, size_t smem, int* occ)
{
    const auto key = std::make_pair(func, smem * 2048 + (size_t)nthr);
    auto it = c->occ_cache.find(key);
    if (it != c->occ_cache.end()) { if (occ) *occ = it->second; return cudaSuccess; }
    {
        std::lock_guard<std::mutex> lock(g_func_mutex);
        size_t& cur = g_func_smem[std::make_pair(c->device, func)];
        if (smem > cur && smem > 32 * 1024) {      // (static shared memory counts against the 48 KB default too)
            cudaError_t e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
            cur = smem;
        }
    }
    int o = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, func, nthr, smem);
    if (e != cudaSuccess) return e;
    if (o < 1) return cudaErrorInvalidConfiguration;
    c->occ_cache[key] = o;
    if (occ) *occ = o;
    return cudaSuccess;
}

#define CK(call)                                                                                        \
    do {                                                                                                \
        cudaError_t e_ = (call);                                                                        \
        if (e_ != cudaSuccess) {                                                                        \
            char buf_[512];                                                                             \
            snprintf(buf_, sizeof buf_, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
            *errp = buf_;                                                                               \
            return (e_ == cudaErrorMemoryAllocation) ? MSD_ENOMEM : MSD_ECUDA;                          \
        }                                                                                               \
    } while (0)

template <class T> static cudaError_t upload(T** d, const T* h, size_t n, cudaStream_t st)
{
    cudaError_t e = cudaMalloc((void**)d, std::max<size_t>(n, 1) * sizeof(T));
    if (e != cudaSuccess) return e;
    if (n) e = cudaMemcpyAsync(*d, h, n * sizeof(T), cudaMemcpyHostToDevice, st);
    return e;
}

static int fail(std::string* errp, int code, const char* msg) { *errp = msg; return code; }

// ---------------------------------------------------------------------------------------------
// setup
// ---------------------------------------------------------------------------------------------
static int do_setup(msd_ctx* c, std::string* errp, int N, int na, int nb, int n_chol, int64_t n_det, const double* h1,
                    const double* L, double e0, const int32_t* occ_ref_a, const int32_t* occ_ref_b,
                    const int64_t* off_a, const int32_t* holes_a, const int32_t* parts_a, const int64_t* off_b,
                    const int32_t* holes_b, const int32_t* parts_b, const double* ci, cudaStream_t st, int shard_rank,
                    int shard_world)
{
    if (shard_world < 1 || shard_rank < 0 || shard_rank >= shard_world) return fail(errp, MSD_EINVAL, "bad determinant shard");
    if (!h1 || !L || !off_a || !off_b || !ci || (na > 0 && !occ_ref_a) || (nb > 0 && !occ_ref_b))
        return fail(errp, MSD_EINVAL, "null pointer argument");
    if (N < 1 || na < 0 || nb < 0 || n_chol < 1 || n_det < 1) return fail(errp, MSD_EINVAL, "non-positive size");
    if (N > 1024 || na > MSD_MAX_NOCC || nb > MSD_MAX_NOCC || na > N || nb > N)
        return fail(errp, MSD_EUNSUPPORTED, "N <= 1024 and n_alpha, n_beta <= 64 required");
    if (n_det >= (int64_t)1 << 31) return fail(errp, MSD_EUNSUPPORTED, "n_det < 2^31 required");
    CK(cudaGetDevice(&c->device));
    CK(cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, c->device));
    c->N = N; c->n_chol = n_chol; c->n_det = n_det; c->e0 = e0;
    const int32_t* occ_ref[2] = {occ_ref_a, occ_ref_b};
    const int64_t* off[2] = {off_a, off_b};
    const int32_t* holes[2] = {holes_a, holes_b};
    const int32_t* parts[2] = {parts_a, parts_b};
    const int ns[2] = {na, nb};

    std::vector<int> pos_in_ref[2];
    int* d_pos_in_ref[2] = {nullptr, nullptr};
    for (int s = 0; s < 2; s++) {
        auto& sp = c->sp[s];
        sp.n = ns[s];
        sp.occ_ref.assign(occ_ref[s], occ_ref[s] + ns[s]);
        pos_in_ref[s].assign(N, -1);
        for (int l = 0; l < ns[s]; l++) {
            int o = sp.occ_ref[l];
            if (o < 0 || o >= N || (l > 0 && o <= sp.occ_ref[l - 1]))
                return fail(errp, MSD_EINVAL, "reference occupation must be strictly ascending and inside [0, N)");
            pos_in_ref[s][o] = l;
        }
        if (off[s][0] != 0) return fail(errp, MSD_EINVAL, "exc_off[0] must be 0");
        CK(upload(&d_pos_in_ref[s], pos_in_ref[s].data(), N, st));
        CK(upload(&sp.d_occ_ref, sp.occ_ref.data(), ns[s], st));
    }
    // --- tables to the device ---
    int64_t* d_off[2]; int32_t* d_holes[2]; int32_t* d_parts[2];
    for (int s = 0; s < 2; s++) {
        int64_t nnz = off[s][n_det];
        if (nnz < 0) return fail(errp, MSD_EINVAL, "negative table size");
        if (nnz > 0 && (!holes[s] || !parts[s])) return fail(errp, MSD_EINVAL, "null table");
        CK(upload(&d_off[s], off[s], (size_t)n_det + 1, st));
        CK(upload(&d_holes[s], holes[s], (size_t)nnz, st));
        CK(upload(&d_parts[s], parts[s], (size_t)nnz, st));
    }
    double* d_ci; CK(upload(&d_ci, ci, (size_t)n_det, st));
    // --- pass 1: validate, mark the active window (reading A10) ---
    int* d_used; CK(cudaMalloc(&d_used, sizeof(int) * (4 * N + 1)));
    CK(cudaMemsetAsync(d_used, 0, sizeof(int) * (4 * N + 1), st));
    int* d_err = d_used + 4 * N;
    for (int s = 0; s < 2; s++) {
        CK(launch_pack_mark(n_det, d_off[s], d_holes[s], d_parts[s], N, d_pos_in_ref[s], d_used + (2 * s) * N,
                            d_used + (2 * s + 1) * N, d_err, st));
        c->launches++;
    }
    std::vector<int> used(4 * N + 1);
    CK(cudaMemcpyAsync(used.data(), d_used, sizeof(int) * (4 * N + 1), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (used[4 * N] != 0) {
        char b[160];
        snprintf(b, sizeof b, "invalid excitation table (error bits 0x%x: 1 range, 2 hole not in reference, "
                 "4 particle in reference, 16 level)", used[4 * N]);
        *errp = b;
        return MSD_EINVAL;
    }
    std::vector<int> map_h[2], map_p[2];
    int* d_map[4];
    for (int s = 0; s < 2; s++) {
        auto& sp = c->sp[s];
        map_h[s].assign(N, -1); map_p[s].assign(N, -1);
        for (int o = 0; o < N; o++) {
            if (used[(2 * s) * N + o]) { map_h[s][o] = (int)sp.act_o.size(); sp.act_o.push_back(o); sp.pos_o.push_back(pos_in_ref[s][o]); }
            if (used[(2 * s + 1) * N + o]) { map_p[s][o] = (int)sp.act_v.size(); sp.act_v.push_back(o); }
        }
        sp.n_o = (int)sp.act_o.size(); sp.n_v = (int)sp.act_v.size();
        sp.n_r = sp.n + sp.n_v; sp.P = sp.n_o * sp.n_v;
        if (sp.n_o > 255 || sp.n_v > 255 || sp.P > 8192)
            return fail(errp, MSD_EUNSUPPORTED, "active window too large (n_o, n_v <= 255, n_o*n_v <= 8192 per spin)");
        if (sp.P > 4096) { c->energy_ok = false; c->energy_why = "local energy requires n_o*n_v <= 4096 per spin"; }
        CK(upload(&d_map[2 * s], map_h[s].data(), N, st));
        CK(upload(&d_map[2 * s + 1], map_p[s].data(), N, st));
        CK(upload(&sp.d_act_v, sp.act_v.data(), sp.act_v.size(), st));
        CK(upload(&sp.d_pos_o, sp.pos_o.data(), sp.pos_o.size(), st));
    }
    {   // the scalar S7 kernel (windows wider than 16 x 16) keeps per-walker tiles in shared memory
        bool mma = true;
        for (int s = 0; s < 2; s++) if (c->sp[s].n > 0 && (c->sp[s].n_o > 16 || c->sp[s].n_v > 16)) mma = false;
        if (!mma && energy_dense_smem(c, 1) > 227 * 1024 && c->energy_ok) {
            c->energy_ok = false;
            c->energy_why = "local energy: n^2 + 2 n n_v + 2 n_o n_v complex numbers per spin must fit in 227 KB of shared memory";
        }
    }
    // --- pass 2: per-determinant rows, phases, level keys ---
    constexpr int NK = (MSD_MAX_LEVEL + 1) * (MSD_MAX_LEVEL + 1);
    unsigned char* d_tmp; int* d_key; double* d_coef_unsorted; int* d_hist;
    CK(cudaMalloc(&d_tmp, (size_t)n_det * 64));
    CK(cudaMalloc(&d_key, sizeof(int) * n_det));
    CK(cudaMalloc(&d_coef_unsorted, sizeof(double) * n_det));
    CK(cudaMalloc(&d_hist, sizeof(int) * NK));
    CK(cudaMemsetAsync(d_hist, 0, sizeof(int) * NK, st));
    CK(launch_pack_rows(n_det, N, d_off[0], d_holes[0], d_parts[0], d_off[1], d_holes[1], d_parts[1],
                        c->sp[0].d_occ_ref, na, c->sp[1].d_occ_ref, nb, d_pos_in_ref[0], d_pos_in_ref[1],
                        d_map[0], d_map[1], d_map[2], d_map[3], d_ci, d_tmp, d_key, d_coef_unsorted, d_hist, d_err, st));
    c->launches++;
    std::vector<int> hist(NK);
    int err2 = 0;
    CK(cudaMemcpyAsync(hist.data(), d_hist, sizeof(int) * NK, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(&err2, d_err, sizeof(int), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (err2 != 0) return fail(errp, MSD_EINVAL, "invalid excitation table (repeated index inside a determinant, or level > n)");
    // --- pass 3: the same determinant listed twice?  (Eq. 15: orthogonal CI expansion) ---
    {
        int64_t nslots = 16;
        while (nslots < 2 * n_det) nslots <<= 1;
        int* d_slots; CK(cudaMalloc(&d_slots, sizeof(int) * nslots));
        CK(cudaMemsetAsync(d_slots, 0xff, sizeof(int) * nslots, st));
        CK(launch_pack_dedup(n_det, d_tmp, d_key, d_slots, nslots, d_err, st));
        c->launches++;
        CK(cudaMemcpyAsync(&err2, d_err, sizeof(int), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        cudaFree(d_slots);
        if (err2 != 0) return fail(errp, MSD_EINVAL, "invalid excitation table (the same determinant is listed twice)");
    }
    // --- buckets ---
    std::vector<int> bucket_keys, bucket_of_key(NK, -1);
    std::vector<int64_t> bucket_start;
    int64_t run = 0, tab_bytes = 0;
    for (int ky = 0; ky < NK; ky++) {
        if (!hist[ky]) continue;
        Bucket b;
        b.ka = ky / (MSD_MAX_LEVEL + 1); b.kb = ky % (MSD_MAX_LEVEL + 1);
        b.start = run; b.count = hist[ky];
        b.rs = std::max(4, (2 * b.ka + 2 * b.kb + 3) / 4 * 4);
        b.tab_off = tab_bytes;
        tab_bytes += (b.count * b.rs + 15) / 16 * 16;
        run += b.count;
        bucket_of_key[ky] = (int)c->buckets.size();
        bucket_keys.push_back(ky);
        bucket_start.push_back(b.start);
        c->buckets.push_back(b);
        c->sp[0].kmax = std::max(c->sp[0].kmax, b.ka);
        c->sp[1].kmax = std::max(c->sp[1].kmax, b.kb);
    }
    if (run != n_det) return fail(errp, MSD_ECUDA, "internal: histogram does not sum to n_det");
    const int nbk = (int)c->buckets.size();
    int* d_bkeys; int64_t* d_bstart; int64_t* d_perm; Bucket* d_buckets; int* d_bok;
    CK(upload(&d_bkeys, bucket_keys.data(), nbk, st));
    CK(upload(&d_bstart, bucket_start.data(), nbk, st));
    CK(upload(&d_buckets, c->buckets.data(), nbk, st));
    CK(upload(&d_bok, bucket_of_key.data(), NK, st));
    CK(cudaMalloc(&d_perm, sizeof(int64_t) * n_det));
    CK(cudaMalloc(&c->d_tab, std::max<int64_t>(tab_bytes, 16)));
    CK(cudaMalloc(&c->d_coef, sizeof(double) * n_det));
    CK(launch_pack_scatter(n_det, d_key, nbk, d_bkeys, d_bstart, d_perm, st));
    CK(launch_pack_write(n_det, d_perm, d_key, d_tmp, d_coef_unsorted, nbk, d_buckets, d_bok, c->d_tab, c->d_coef, st));
    c->launches += 2;
    c->h_perm.resize(n_det); c->h_coef.resize(n_det);
    CK(cudaMemcpyAsync(c->h_perm.data(), d_perm, sizeof(int64_t) * n_det, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(c->h_coef.data(), c->d_coef, sizeof(double) * n_det, cudaMemcpyDeviceToHost, st));
    // --- L_sub, h1_sub (A17): rows occ_ref U act_virt, row stride ldN (even) ---
    const int ldN = N + (N & 1);
    {
        double* d_L; double* d_h1;
        CK(upload(&d_L, L, (size_t)n_chol * N * N, st));
        CK(upload(&d_h1, h1, (size_t)N * N, st));
        for (int s = 0; s < 2; s++) {
            auto& sp = c->sp[s];
            std::vector<int> rows(sp.occ_ref);
            rows.insert(rows.end(), sp.act_v.begin(), sp.act_v.end());
            int* d_rows; CK(upload(&d_rows, rows.data(), rows.size(), st));
            size_t nel = (size_t)(n_chol + 1) * sp.n_r * ldN;
            CK(cudaMalloc(&sp.d_Lsub, std::max<size_t>(nel, 2) * sizeof(double)));
            CK(cudaMemsetAsync(sp.d_Lsub, 0, std::max<size_t>(nel, 2) * sizeof(double), st));
            // packed with row stride ldN: copy N columns of each row
            if (sp.n_r > 0) {
                // reuse the pack kernel with "N" = source stride; destination stride handled by a 2D copy
                double* tmp; CK(cudaMalloc(&tmp, (size_t)(n_chol + 1) * sp.n_r * N * sizeof(double)));
                CK(launch_pack_lsub(d_L, n_chol, N, sp.n_r, d_rows, tmp, st));
                CK(launch_pack_lsub(d_h1, 1, N, sp.n_r, d_rows, tmp + (size_t)n_chol * sp.n_r * N, st));
                c->launches += 2;
                CK(cudaMemcpy2DAsync(sp.d_Lsub, ldN * sizeof(double), tmp, N * sizeof(double), N * sizeof(double),
                                     (size_t)(n_chol + 1) * sp.n_r, cudaMemcpyDeviceToDevice, st));
                CK(cudaStreamSynchronize(st));
                cudaFree(tmp);
            }
            CK(cudaStreamSynchronize(st));
            cudaFree(d_rows);
        }
        cudaFree(d_L); cudaFree(d_h1);
    }
    CK(cudaStreamSynchronize(st));
    c->h_ka.resize(n_det); c->h_kb.resize(n_det);
    for (const Bucket& b : c->buckets)
        for (int64_t i = 0; i < b.count; i++) { c->h_ka[b.start + i] = b.ka; c->h_kb[b.start + i] = b.kb; }
    // --- work items ---
    for (const Bucket& b : c->buckets)
        if (b.ka * b.ka + b.kb * b.kb > 400) return fail(errp, MSD_EUNSUPPORTED, "k_alpha^2 + k_beta^2 <= 400 required");
    // Determinant sharding: this context evaluates slice shard_rank of shard_world of EVERY level
    // bucket (so that all ranks get the same level mix); the window, the table and the introspection stay those of the whole
    // trial.  `work` are the buckets the work items are cut from.
    c->shard_rank = shard_rank; c->shard_world = shard_world;
    std::vector<Bucket> work(c->buckets);
    for (Bucket& b : work) {
        const int64_t lo = b.count * shard_rank / shard_world, hi = b.count * (shard_rank + 1) / shard_world;
        b.start += lo; b.tab_off += lo * b.rs; b.count = hi - lo;
    }
    auto cost = [](int ka, int kb) {
        double a = ka, b = kb;
        return 1.0 + a * a * a + b * b * b + a * a * b * b;
    };
    auto cls = [](const WorkItem& w) { int m = std::max(w.ka, w.kb); return m <= 2 ? 0 : (m == 3 ? 1 : 2); };
    static const int gen_thresholds[] = {26, 34, 41, 50, 72, 100, 128, 162, 200, 400};
    auto grp = [](const WorkItem& w) {
        int e = w.ka * w.ka + w.kb * w.kb, g = 0;
        while (gen_thresholds[g] < e) g++;
        return g;
    };
    for (int bi = 0; bi < nbk; bi++) {
        const Bucket& b = work[bi];
        const bool gen = std::max(b.ka, b.kb) > MSD_CF_MAX;
        const int m = std::max(b.ka, b.kb);
        int slots = gen ? 128 / MSD_WT : (m <= 3 ? 256 : 128) / MSD_WT;
        int iters = (int)std::max(4.0, std::min(32.0, 1024.0 / cost(b.ka, b.kb)));
        if (gen) iters = (int)std::max(1.0, std::min(4.0, 1024.0 / cost(b.ka, b.kb)));   // few, heavy determinants: more CTAs
        int dpc = slots * iters;
        for (int64_t i0 = 0; i0 < b.count; i0 += dpc) {
            WorkItem it;
            it.bucket = bi; it.ka = b.ka; it.kb = b.kb; it.rs = b.rs;
            it.det_begin = b.start + i0;
            it.det_count = (int)std::min<int64_t>(dpc, b.count - i0);
            it.tab_off = b.tab_off + i0 * b.rs;
            (gen ? c->items_gen : c->items_cf).push_back(it);
        }
    }
    auto icost = [&](const WorkItem& w) { return cost(w.ka, w.kb) * w.det_count; };
    std::stable_sort(c->items_cf.begin(), c->items_cf.end(), [&](const WorkItem& x, const WorkItem& y) {
        if (cls(x) != cls(y)) return cls(x) < cls(y);
        return icost(x) > icost(y);
    });
    std::stable_sort(c->items_gen.begin(), c->items_gen.end(), [&](const WorkItem& x, const WorkItem& y) {
        if (grp(x) != grp(y)) return grp(x) < grp(y);
        return icost(x) > icost(y);
    });
    for (int cl = 0; cl <= 3; cl++) {
        int i = 0;
        while (i < (int)c->items_cf.size() && cls(c->items_cf[i]) < cl) i++;
        c->cf_class_begin[cl] = i;
    }
    c->gen_group_begin.clear(); c->gen_group_elems.clear();
    for (int g = 0; g <= 10; g++) {
        int i = 0;
        while (i < (int)c->items_gen.size() && grp(c->items_gen[i]) < g) i++;
        c->gen_group_begin.push_back(i);
        if (g < 10) c->gen_group_elems.push_back(gen_thresholds[g]);
    }
    // Owner-pull lists of the force-bias CI reduction (msd_internal.cuh PULL_*)
    {
        const int noa = c->sp[0].n_o, nob = c->sp[1].n_o, Pa = c->sp[0].P, PT = c->sp[0].P + c->sp[1].P;
        // shared memory beside the C tile (and the g tile when it fits as well): scale factors + staged adjugates
        // layout (bytes from the start of dynamic shared memory): C tile | 16 B holding 1.0 | pool | g tile
        const size_t tile_bytes = (size_t)PT * MSD_WT * sizeof(cplx), total = 225 * 1024;
        size_t per_det_max = 256;
        for (const Bucket& b : c->buckets)
            if (std::max(b.ka, b.kb) <= MSD_CF_MAX)
                per_det_max = std::max<size_t>(per_det_max, 256 + (size_t)((b.ka >= 3 ? b.ka * b.ka : 0) + (b.kb >= 3 ? b.kb * b.kb : 0)) * 128);
        // the g tile must sit in shared memory (level-2 entries address it directly) and every bucket needs >= 16 determinants
        c->pull_gs = true;
        c->pull_pool = (2 * tile_bytes + 16 * per_det_max + 256 <= total) ? total - 2 * tile_bytes - 256 : 0;
        if (PT >= (1 << 14)) c->pull_pool = 0;
        int64_t tab_bytes_all = 0;
        for (const Bucket& b : c->buckets) tab_bytes_all = std::max<int64_t>(tab_bytes_all, b.tab_off + (b.count * b.rs + 15) / 16 * 16);
        std::vector<unsigned char> htab((size_t)std::max<int64_t>(tab_bytes_all, 16));
        CK(cudaMemcpyAsync(htab.data(), c->d_tab, (size_t)tab_bytes_all, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        auto pcls = [](const WorkItem& w) { return std::max(w.ka, w.kb) <= 3 ? 0 : 1; };
        auto estage = [](int ka, int kb) { return (ka >= 3 ? ka * ka : 0) + (kb >= 3 ? kb * kb : 0); };
        for (int bi = 0; bi < nbk && c->pull_pool; bi++) {
            const Bucket& b = work[bi];
            if (std::max(b.ka, b.kb) > MSD_CF_MAX) continue;
            const int slots = (std::max(b.ka, b.kb) <= 3 ? 512 : 256) / MSD_WT;
            int D = (int)std::min<size_t>(PULL_DMAX, c->pull_pool / (256 + (size_t)estage(b.ka, b.kb) * 128));
            if (D > slots) D = D / slots * slots;                 // whole sweeps of the CTA's determinant slots
            for (int64_t i0 = 0; i0 < b.count; i0 += D) {
                WorkItem it;
                it.bucket = bi; it.ka = b.ka; it.kb = b.kb; it.rs = b.rs;
                it.det_begin = b.start + i0;
                it.det_count = (int)std::min<int64_t>(D, b.count - i0);
                it.tab_off = b.tab_off + i0 * b.rs;
                it.sched_off = 0; it.pull_off = 0;
                c->items_pull.push_back(it);
            }
        }
        // by class, heaviest chunks first (the persistent CTAs take them in snake order)
        std::stable_sort(c->items_pull.begin(), c->items_pull.end(), [&](const WorkItem& x, const WorkItem& y) {
            if (pcls(x) != pcls(y)) return pcls(x) < pcls(y);
            auto w = [](const WorkItem& t) {
                auto f = [](int k) { return k <= 1 ? 2.0 : (k == 2 ? 20.0 : (k == 3 ? 160.0 : 600.0)); };
                return (f(t.ka) + f(t.kb) + 10.0 * (t.ka * t.ka + t.kb * t.kb) + 30.0) * t.det_count;
            };
            return w(x) > w(y);
        });
        for (int cl = 0; cl <= 2; cl++) {
            int i = 0;
            while (i < (int)c->items_pull.size() && pcls(c->items_pull[i]) < cl) i++;
            c->pull_class_begin[cl] = i;
        }
        std::vector<unsigned short> splits;
        std::vector<uint2> ents;
        std::vector<uint32_t> cnt((size_t)PT + 1);
        for (size_t ii = 0; ii < c->items_pull.size(); ii++) {
            WorkItem& w = c->items_pull[ii];
            const int G = (pcls(w) == 0 ? 512 : 256) / MSD_WT;
            w.pull_off = (int64_t)splits.size();
            w.sched_off = (int64_t)ents.size();
            const int ka = w.ka, kb = w.kb;
            const uint32_t one_off = (uint32_t)tile_bytes, pool_off = (uint32_t)tile_bytes + 256u;
            const uint32_t stage_off = pool_off + (uint32_t)w.det_count * 256u, g_off = pool_off + (uint32_t)c->pull_pool;
            std::fill(cnt.begin(), cnt.end(), 0u);
            auto xof = [&](const unsigned char* row, int s, int a, int b) -> uint32_t {
                return s == 0 ? (uint32_t)row[ka + b] * noa + row[a]
                              : (uint32_t)Pa + (uint32_t)row[2 * ka + kb + b] * nob + row[2 * ka + a];
            };
            for (int d = 0; d < w.det_count; d++) {
                const unsigned char* row = htab.data() + w.tab_off + (int64_t)d * w.rs;
                for (int s = 0; s < 2; s++) {
                    const int k = s ? kb : ka;
                    for (int a = 0; a < k; a++) for (int b = 0; b < k; b++) cnt[xof(row, s, a, b) + 1]++;
                }
            }
            for (int x = 0; x < PT; x++) cnt[x + 1] += cnt[x];
            const uint32_t n_ent = cnt[PT];
            // piece boundaries: the first change of x at or after q * n / G
            {
                int x = 0;
                for (int q = 0; q <= G; q++) {
                    const uint32_t target = (uint32_t)(((uint64_t)n_ent * q + G - 1) / G);
                    while (x < PT && cnt[x] < target) x++;
                    splits.push_back((unsigned short)(q == G ? n_ent : cnt[x]));
                }
            }
            const size_t base = ents.size();
            ents.resize(base + n_ent);
            for (int d = 0; d < w.det_count; d++) {
                const unsigned char* row = htab.data() + w.tab_off + (int64_t)d * w.rs;
                for (int s = 0; s < 2; s++) {
                    const int k = s ? kb : ka, no = s ? nob : noa;
                    const unsigned char* h = row + (s ? 2 * ka : 0);
                    const unsigned char* pp = h + k;
                    const int eoff = (s && ka >= 3) ? ka * ka : 0;
                    for (int a = 0; a < k; a++)
                        for (int b = 0; b < k; b++) {
                            const uint32_t x = xof(row, s, a, b);
                            // w1 = byte offset (walker 0) of the value the entry multiplies: the constant 1.0, an element of the
                            // g tile, or an element of the staged adjugate (which carries its own sign)
                            uint32_t w1, sign = (uint32_t)((a + b) & 1);
                            if (k == 1) { w1 = one_off; sign = 0; }
                            else if (k == 2) w1 = g_off + ((s ? (uint32_t)Pa : 0u) + (uint32_t)pp[1 - b] * no + h[1 - a]) * 128u;
                            else { w1 = stage_off + (uint32_t)((eoff + a * k + b) * w.det_count + d) * 128u; sign = 0; }
                            // w0 = (2 det + spin) [10 bits: byte offset / 128 of the scale factor] | sign << 10 | x << 11 | last << 25
                            ents[base + cnt[x]++] = make_uint2((uint32_t)(2 * d + s) | sign << 10 | x << 11, w1);
                        }
                }
            }
            for (uint32_t t = 0; t < n_ent; t++)      // last entry of every x-run
                if (t + 1 == n_ent || ((ents[base + t].x >> 11) & 0x3fffu) != ((ents[base + t + 1].x >> 11) & 0x3fffu))
                    ents[base + t].x |= 1u << 25;
        }
        if (splits.empty()) splits.push_back(0);
        if (ents.empty()) ents.push_back(make_uint2(0u, 0u));
        CK(upload(&c->d_pull_off, splits.data(), splits.size(), st));
        CK(upload(&c->d_pull_ent, ents.data(), ents.size(), st));
        CK(upload(&c->d_items_pull, c->items_pull.data(), c->items_pull.size(), st));
        CK(cudaStreamSynchronize(st));
    }
    {
        int a, b, m, t, ko, kv;
        c->need_lam = !energy_fused_shape(c, &a, &b, &m, &t, &ko, &kv);
    }
    CK(upload(&c->d_items_cf, c->items_cf.data(), c->items_cf.size(), st));
    CK(upload(&c->d_items_gen, c->items_gen.data(), c->items_gen.size(), st));
    CK(cudaStreamSynchronize(st));
    // free setup temporaries
    for (int s = 0; s < 2; s++) { cudaFree(d_pos_in_ref[s]); cudaFree(d_off[s]); cudaFree(d_holes[s]); cudaFree(d_parts[s]); }
    for (int i = 0; i < 4; i++) cudaFree(d_map[i]);
    cudaFree(d_ci); cudaFree(d_used); cudaFree(d_tmp); cudaFree(d_key); cudaFree(d_coef_unsorted); cudaFree(d_hist);
    cudaFree(d_bkeys); cudaFree(d_bstart); cudaFree(d_perm); cudaFree(d_buckets); cudaFree(d_bok);
    return MSD_OK;
}

extern "C" int msd_setup(msd_ctx** out, int N, int n_alpha, int n_beta, int n_chol, int64_t n_det, const double* h1,
                         const double* L, double e0, const int32_t* occ_ref_a, const int32_t* occ_ref_b,
                         const int64_t* exc_off_a, const int32_t* holes_a, const int32_t* parts_a,
                         const int64_t* exc_off_b, const int32_t* holes_b, const int32_t* parts_b, const double* ci,
                         void* stream)
{
    return msd_setup_sharded(out, N, n_alpha, n_beta, n_chol, n_det, h1, L, e0, occ_ref_a, occ_ref_b, exc_off_a, holes_a, parts_a,
                             exc_off_b, holes_b, parts_b, ci, 0, 1, stream);
}

extern "C" int msd_setup_sharded(msd_ctx** out, int N, int n_alpha, int n_beta, int n_chol, int64_t n_det, const double* h1,
                                 const double* L, double e0, const int32_t* occ_ref_a, const int32_t* occ_ref_b,
                                 const int64_t* exc_off_a, const int32_t* holes_a, const int32_t* parts_a,
                                 const int64_t* exc_off_b, const int32_t* holes_b, const int32_t* parts_b, const double* ci,
                                 int shard_rank, int shard_world, void* stream)
{
    if (!out) { g_setup_error = "out is NULL"; return MSD_EINVAL; }
    *out = nullptr;
    msd_ctx* c = new (std::nothrow) msd_ctx();
    if (!c) { g_setup_error = "out of host memory"; return MSD_ENOMEM; }
    std::string err;
    int rc;
    try {
        rc = do_setup(c, &err, N, n_alpha, n_beta, n_chol, n_det, h1, L, e0, occ_ref_a, occ_ref_b, exc_off_a, holes_a,
                      parts_a, exc_off_b, holes_b, parts_b, ci, (cudaStream_t)stream, shard_rank, shard_world);
    } catch (const std::bad_alloc&) {
        rc = MSD_ENOMEM; err = "out of host memory";
    }
    if (rc != MSD_OK) {
        g_setup_error = err;
        cudaGetLastError();
        msd_destroy(c);
        return rc;
    }
    *out = c;
    return MSD_OK;
}

extern "C" int msd_setup_from_occ(msd_ctx** out, int N, int n_alpha, int n_beta, int n_chol, int64_t n_det,
                                  const double* h1, const double* L, double e0, const int32_t* occa,
                                  const int32_t* occb, const double* ci, void* stream)
{
    if (!out || n_det < 1 || N < 1 || n_alpha < 0 || n_beta < 0 || (n_alpha > 0 && !occa) || (n_beta > 0 && !occb)) {
        g_setup_error = "bad argument";
        return MSD_EINVAL;
    }
    // pure set bookkeeping on the host: reference = sorted row 0; holes = ref \ occ, particles = occ \ ref
    try {
        std::vector<int32_t> ref[2];
        std::vector<int64_t> off[2];
        std::vector<int32_t> holes[2], parts[2];
        const int32_t* occ[2] = {occa, occb};
        const int ns[2] = {n_alpha, n_beta};
        for (int s = 0; s < 2; s++) {
            ref[s].assign(occ[s], occ[s] + ns[s]);
            std::sort(ref[s].begin(), ref[s].end());
            std::vector<char> inref(N, 0), inocc(N, 0);
            for (int o : ref[s]) { if (o < 0 || o >= N) { g_setup_error = "orbital out of range"; return MSD_EINVAL; } inref[o] = 1; }
            off[s].assign(n_det + 1, 0);
            for (int64_t I = 0; I < n_det; I++) {
                const int32_t* row = occ[s] + I * ns[s];
                for (int l = 0; l < ns[s]; l++) {
                    if (row[l] < 0 || row[l] >= N) { g_setup_error = "orbital out of range"; return MSD_EINVAL; }
                    if (inocc[row[l]]) { g_setup_error = "repeated orbital in an occupation list"; return MSD_EINVAL; }
                    inocc[row[l]] = 1;
                    if (!inref[row[l]]) parts[s].push_back(row[l]);
                }
                for (int o : ref[s]) if (!inocc[o]) holes[s].push_back(o);
                for (int l = 0; l < ns[s]; l++) inocc[row[l]] = 0;
                off[s][I + 1] = (int64_t)parts[s].size();
                if (holes[s].size() != parts[s].size()) { g_setup_error = "internal: hole/particle mismatch"; return MSD_EINVAL; }
            }
        }
        return msd_setup(out, N, n_alpha, n_beta, n_chol, n_det, h1, L, e0, ref[0].data(), ref[1].data(),
                         off[0].data(), holes[0].data(), parts[0].data(), off[1].data(), holes[1].data(),
                         parts[1].data(), ci, stream);
    } catch (const std::bad_alloc&) {
        g_setup_error = "out of host memory";
        return MSD_ENOMEM;
    }
}

extern "C" void msd_destroy(msd_ctx* c)
{
    if (!c) return;
    for (int s = 0; s < 2; s++) {
        cudaFree(c->sp[s].d_occ_ref); cudaFree(c->sp[s].d_act_v); cudaFree(c->sp[s].d_pos_o); cudaFree(c->sp[s].d_Lsub);
    }
    cudaFree(c->d_tab); cudaFree(c->d_coef); cudaFree(c->d_items_cf); cudaFree(c->d_items_gen);
    cudaFree(c->d_items_pull); cudaFree(c->d_pull_off); cudaFree(c->d_pull_ent);
    cudaFree(c->d_LT); cudaFree(c->d_hp); cudaFree(c->d_E);
    cudaFree(c->ws.base);
    cudaFree(c->stg_a); cudaFree(c->stg_b); cudaFree(c->stg_out); cudaFree(c->stg_flags);
    for (auto& e : c->ev) if (e) cudaEventDestroy(e);
    for (auto& a : c->aux) if (a) cudaStreamDestroy(a);
    for (auto& e : c->ev_join) if (e) cudaEventDestroy(e);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_done) cudaEventDestroy(c->ev_done);
    delete c;
}

extern "C" const char* msd_last_error(const msd_ctx* c) { return c ? c->err.c_str() : g_setup_error.c_str(); }

extern "C" int msd_get_info(const msd_ctx* c, int64_t* info)
{
    if (!c || !info) return MSD_EINVAL;
    info[0] = c->sp[0].n_o; info[1] = c->sp[0].n_v; info[2] = c->sp[1].n_o; info[3] = c->sp[1].n_v;
    info[4] = (int64_t)c->buckets.size(); info[5] = c->sp[0].kmax; info[6] = c->sp[1].kmax; info[7] = MSD_WT;
    info[8] = c->energy_ok ? 1 : 0;
    info[9] = c->shard_rank; info[10] = c->shard_world;
    return MSD_OK;
}

extern "C" int msd_get_packed(const msd_ctx* c, int64_t* perm, double* coef, int32_t* la, int32_t* lb)
{
    if (!c) return MSD_EINVAL;
    if (perm) memcpy(perm, c->h_perm.data(), sizeof(int64_t) * c->n_det);
    if (coef) memcpy(coef, c->h_coef.data(), sizeof(double) * c->n_det);
    if (la) memcpy(la, c->h_ka.data(), sizeof(int32_t) * c->n_det);
    if (lb) memcpy(lb, c->h_kb.data(), sizeof(int32_t) * c->n_det);
    return MSD_OK;
}

extern "C" int msd_set_workspace_limit(msd_ctx* c, int64_t bytes)
{
    if (!c || bytes < 0) return MSD_EINVAL;
    c->ws_limit = bytes;
    c->ws_limit_auto = 0;        // re-read the free memory at the next call
    c->ws.want = 0;              // and lay the workspace out again (the fast path of ensure_workspace keys on it)
    return MSD_OK;
}
extern "C" int msd_set_allreduce(msd_ctx* c, msd_allreduce_fn fn, void* user)
{
    if (!c) return MSD_EINVAL;
    c->allreduce = fn; c->allreduce_user = user;
    return MSD_OK;
}
extern "C" int msd_set_option(msd_ctx* c, int option, int64_t value)
{
    if (!c) return MSD_EINVAL;
    if (option == MSD_OPT_NO_SMEM_TILES && value >= 0 && value <= 2) { c->no_smem_tiles = (int)value; return MSD_OK; }
    if (option == MSD_OPT_NO_3M && (value == 0 || value == 1)) { c->no_3m = value != 0; return MSD_OK; }
    if (option == MSD_OPT_3M_MAX_COND && value >= 0) { c->v3m_max_cond = (double)value; return MSD_OK; }
    if (option == MSD_OPT_COOP_MIN_ELEMS && value >= 0 && value <= 200) { c->coop_min_elems = c->coop_min_elems_fb = (int)value; return MSD_OK; }
    if (option == MSD_OPT_NO_FUSED_S7 && (value == 0 || value == 1)) {
        c->no_fused = value != 0;
        int a, b, m, t, ko, kv;
        c->need_lam = c->no_fused || !energy_fused_shape(c, &a, &b, &m, &t, &ko, &kv);
        c->ws.want = 0;                  // the workspace layout changes (Lambda buffer)
        return MSD_OK;
    }
    c->err = "unknown option or value";
    return MSD_EINVAL;
}
extern "C" int64_t msd_launch_count(const msd_ctx* c) { return c ? c->launches : -1; }
extern "C" int msd_set_profiling(msd_ctx* c, int on)
{
    if (!c) return MSD_EINVAL;
    c->profiling = on != 0;
    if (c->profiling)
        for (auto& e : c->ev) if (!e && cudaEventCreate(&e) != cudaSuccess) return MSD_ECUDA;
    return MSD_OK;
}
extern "C" int msd_get_phase_ms(msd_ctx* c, float* ms, int n)
{
    if (!c || !ms) return MSD_EINVAL;
    for (int i = 0; i < n && i < 6; i++) ms[i] = c->phase_ms[i];
    return MSD_OK;
}

// ---------------------------------------------------------------------------------------------
// fork/join over the context's side streams
// ---------------------------------------------------------------------------------------------
cudaStream_t Fork::stream(int i)
{
    if (err != cudaSuccess) return st;
    const int a = (i - 1) % msd_ctx::NAUX;
    if (!c->ev_fork) {
        if ((err = cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming)) != cudaSuccess) return st;
        for (int k = 0; k < msd_ctx::NAUX; k++) {
            if ((err = cudaStreamCreateWithFlags(&c->aux[k], cudaStreamNonBlocking)) != cudaSuccess) return st;
            if ((err = cudaEventCreateWithFlags(&c->ev_join[k], cudaEventDisableTiming)) != cudaSuccess) return st;
        }
    }
    if (!forked) {
        if ((err = cudaEventRecord(c->ev_fork, st)) != cudaSuccess) return st;
        forked = true;       // the fork point precedes every launch of the group, also those on st itself
    }
    if (i <= 0) return st;
    if (!(used & (1 << a))) {
        if ((err = cudaStreamWaitEvent(c->aux[a], c->ev_fork, 0)) != cudaSuccess) return st;
        used |= 1 << a;
    }
    return c->aux[a];
}

cudaError_t Fork::join()
{
    for (int a = 0; a < msd_ctx::NAUX && err == cudaSuccess; a++) {
        if (!(used & (1 << a))) continue;
        if ((err = cudaEventRecord(c->ev_join[a], c->aux[a])) != cudaSuccess) break;
        err = cudaStreamWaitEvent(st, c->ev_join[a], 0);
    }
    used = 0; forked = false;
    return err;
}

// ---------------------------------------------------------------------------------------------
// workspace
// ---------------------------------------------------------------------------------------------
struct Carver {
    char* base; size_t off = 0;
    explicit Carver(char* b) : base(b) {}
    template <class T> T* take(size_t n) {
        off = (off + 255) / 256 * 256;
        T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
        off += std::max<size_t>(n, 1) * sizeof(T);
        return p;
    }
};

// lays the workspace out for wc walkers at `level`; with base == nullptr only measures
static size_t carve(const msd_ctx* c, Workspace& ws, char* base, int64_t wc, int level)
{
    Carver k(base);
    const int N = c->N, ldN = N + (N & 1), ng = c->n_chol;
    const int64_t nt = wc / MSD_WT;
    // zero region first
    char* z0 = base ? base : nullptr;
    for (int s = 0; s < 2; s++) ws.C[s] = k.take<double>((size_t)nt * c->sp[s].P * 2 * MSD_WT);
    ws.Wacc = k.take<cplx>(wc);
    ws.E2nd = k.take<cplx>(wc);
    ws.E1nd = k.take<cplx>(wc);
    ws.wflags = k.take<int>(wc);
    if (level == 3) {
        for (int s = 0; s < 2; s++) ws.F[s] = k.take<cplx>((size_t)wc * c->sp[s].P);
        ws.Eacc = k.take<cplx>((size_t)wc * 2);
    }
    if (level == 3) ws.X0 = k.take<cplx>((size_t)2 * wc * ng);   // zero for a spin without electrons
    k.off = (k.off + 255) / 256 * 256;
    ws.zero_begin = z0;
    ws.zero_bytes = k.off;
    for (int s = 0; s < 2; s++) {
        ws.theta[s] = k.take<cplx>((size_t)wc * N * c->sp[s].n);
        ws.g[s] = k.take<cplx>((size_t)nt * c->sp[s].P * MSD_WT);
    }
    ws.det0 = k.take<cplx>((size_t)wc * 2);
    ws.kappa2 = k.take<double>((size_t)wc * 2);
    if (level == 2 || level == 4) {
        for (int s = 0; s < 2; s++) ws.Gp[s] = k.take<double>((size_t)wc * 2 * c->sp[s].n_r * ldN);
    }
    if (level == 4) {
        const int ldg = ng + (ng & 1);
        ws.fbuf = k.take<cplx>((size_t)wc * ng);
        ws.Yf = k.take<double>((size_t)2 * wc * ldg);
        ws.Aw = k.take<cplx>((size_t)wc * N * N);
        ws.ov_old = k.take<cplx>(wc); ws.ov_new = k.take<cplx>(wc); ws.expo = k.take<cplx>(wc);
        ws.fl_old = k.take<int>(wc);
    }
    if (level == 3) {
        for (int s = 0; s < 2; s++) {
            const auto& sp = c->sp[s];
            ws.thetaT[s] = k.take<double>((size_t)wc * sp.n * 2 * ldN);
            ws.Lam[s] = c->need_lam ? k.take<cplx>((size_t)(ng + 1) * sp.n_r * wc * sp.n) : nullptr;
            ws.Bp[s] = k.take<cplx>((size_t)wc * sp.P * ng);
            ws.Vss[s] = k.take<cplx>((size_t)nt * sp.P * sp.P * MSD_WT);
            ws.Hrot[s] = k.take<cplx>((size_t)wc * sp.P);
            ws.FH[s] = k.take<cplx>((size_t)nt * sp.P * 2 * MSD_WT);
        }
        ws.Vab = k.take<cplx>((size_t)nt * c->sp[0].P * c->sp[1].P * MSD_WT);
    }
    return k.off + 256;
}

// level: 1 overlap, 2 force bias / greens, 3 energy, 4 propagation step.  A separate workspace layout per level (the buffers differ);
// reallocated only when the level or the walker capacity changes.
static int ensure_workspace(msd_ctx* c, int level, int64_t nw, std::string* errp)
{
    int64_t want = (nw + MSD_WT - 1) / MSD_WT * MSD_WT;
    if (want == 0) want = MSD_WT;
    Workspace& ws = c->ws;
    if (ws.base && ws.level == level && ws.want == want) return MSD_OK;     // fast path: no CUDA call at all
    int64_t limit = c->ws_limit;
    if (limit == 0) {
        if (c->ws_limit_auto == 0) {
            size_t fr = 0, tot = 0;
            CK(cudaMemGetInfo(&fr, &tot));
            c->ws_limit_auto = (int64_t)((fr + ws.bytes) * 0.7);
        }
        limit = c->ws_limit_auto;
    }
    Workspace probe;
    int64_t wc = want;
    while (wc > MSD_WT && (int64_t)carve(c, probe, nullptr, wc, level) > limit) wc = (wc / 2 + MSD_WT - 1) / MSD_WT * MSD_WT;
    size_t need = carve(c, probe, nullptr, wc, level);
    if ((int64_t)need > limit) return fail(errp, MSD_ENOMEM, "workspace for one walker tile exceeds the limit");
    if (ws.base && ws.bytes >= need) {
        // re-carve inside the existing allocation
        ws.level = level; ws.wc = wc; ws.want = want;
        carve(c, ws, ws.base, wc, level);
        return MSD_OK;
    }
    if (ws.base) { CK(cudaDeviceSynchronize()); cudaFree(ws.base); ws.base = nullptr; ws.bytes = 0; }
    char* p = nullptr;
    CK(cudaMalloc(&p, need));
    ws.base = p; ws.bytes = need; ws.level = level; ws.wc = wc; ws.want = want;
    carve(c, ws, ws.base, wc, level);
    return MSD_OK;
}

// ---------------------------------------------------------------------------------------------
// hot calls
// ---------------------------------------------------------------------------------------------
enum { CALL_OVERLAP = 1, CALL_FB = 2, CALL_GREENS = 4, CALL_ENERGY = 8, CALL_FB_ENERGY = 16, CALL_PROPAGATE = 32, CALL_COND = 64 };

// msd_reference_cond: sqrt of the (||O0||_F ||O0^-1||_F)^2 that k_reference leaves per walker and spin
__global__ void k_cond_out(int64_t n2, const double* __restrict__ kappa2, double* __restrict__ out)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n2) out[i] = sqrt(kappa2[i]);
}

static void mark(msd_ctx* c, int i, cudaStream_t st) { if (c->profiling) cudaEventRecord(c->ev[i], st); }

// Determinant sharding: after a determinant pass the per-walker partial sums of this rank -- C^alpha, C^beta, W, E2nd, E1nd,
// one contiguous run of doubles at the start of the workspace -- are summed over the ranks by the caller's hook (one
// all-reduce of (2 + 2 n_o n_v ...) complex per walker: SURVEY.md 8(e)(ii)) before anything divides by W.
static void shard_reduce(msd_ctx* c, Workspace& ws, cudaStream_t st)
{
    if (!c->allreduce) return;
    const int64_t n = (int64_t)((reinterpret_cast<char*>(ws.E1nd + ws.wc) - reinterpret_cast<char*>(ws.C[0])) / sizeof(double));
    // the partial sums are complete on the device when the hook runs (the determinant kernels ran on forked side streams);
    // a sharded call is a collective anyway, so the host wait costs nothing that the all-reduce does not
    cudaStreamSynchronize(st);
    c->allreduce(c->allreduce_user, ws.C[0], n, (void*)st);
}

// S6: fb[w][g] += sum_(r,q) L_sub^s[g][(r,q)] G^s_w[(r,q)]  (one spin; fb zeroed by the caller: split-K partial sums meet in RED)
static cudaError_t launch_fb_gemm(msd_ctx* c, int s, int64_t nw, Workspace& ws, cplx* fb, cudaStream_t st)
{
    const auto& sp = c->sp[s];
    const int N = c->N, ldN = N + (N & 1), ng = c->n_chol;
    GemmArgs a;
    a.A = sp.d_Lsub; a.B = ws.Gp[s]; a.C = reinterpret_cast<double*>(fb);
    a.M = ng; a.N = (int)(2 * nw); a.K = sp.n_r * ldN;
    a.lda = (int64_t)sp.n_r * ldN; a.ldb = (int64_t)sp.n_r * ldN;
    a.strideA = 0; a.strideB = 0; a.batch = 1;
    a.zdiv = 1; a.strideC_hi = 0; a.strideC_lo = 0; a.cs_m = 1; a.cs_j = ng;
    // skinny output (n_chol x 2 n_w): split K over the SMs, partial sums meet in RED.ADD.F64
    a.accumulate = 2;
    const int64_t tiles = (int64_t)((a.M + 63) / 64) * ((a.N + 63) / 64);
    const int ks = (int)std::max<int64_t>(1, (2 * c->n_sm + tiles - 1) / tiles);
    a.ksplit = std::min(ks, std::max(1, a.K / 64));
    cudaError_t e = launch_gemm_tn(c, a, st);
    c->launches++;
    return e;
}

static int run_chunks(msd_ctx* c, std::string* errp, int call, int64_t n_w, const cplx* phi_a, const cplx* phi_b,
                      cplx* out, int* flags, cudaStream_t st)
{
    const bool energy_like = (call == CALL_ENERGY || call == CALL_FB_ENERGY);
    const int level = (call == CALL_OVERLAP || call == CALL_COND) ? 1 : (energy_like ? 3 : (call == CALL_PROPAGATE ? 4 : 2));
    if (energy_like && !c->energy_ok) return fail(errp, MSD_EUNSUPPORTED, c->energy_why.c_str());
    int rc = ensure_workspace(c, level, n_w, errp);
    if (rc != MSD_OK) return rc;
    // one workspace per context: a call on another stream than the previous call's waits for that call's last kernel
    if (!c->ev_done) CK(cudaEventCreateWithFlags(&c->ev_done, cudaEventDisableTiming));
    if (c->have_done && st != c->last_stream) CK(cudaStreamWaitEvent(st, c->ev_done, 0));
    Workspace& ws = c->ws;
    const int N = c->N, ldN = N + (N & 1), ng = c->n_chol;
    for (int i = 0; i < 6; i++) c->phase_ms[i] = 0.f;
    for (int64_t w0 = 0; w0 < n_w; w0 += ws.wc) {
        const int64_t nw = std::min<int64_t>(ws.wc, n_w - w0);
        const cplx* pa = phi_a + w0 * (int64_t)N * c->sp[0].n;
        const cplx* pb = phi_b + w0 * (int64_t)N * c->sp[1].n;
        int* fl = flags ? flags + w0 : nullptr;
        CK(cudaMemsetAsync(ws.zero_begin, 0, ws.zero_bytes, st));
        mark(c, 0, st);
        CK(launch_reference(c, N, ldN, c->dev(0), c->dev(1), nw, pa, pb, ws, level == 3, st));
        c->launches++;
        mark(c, 1, st);
        if (call == CALL_COND) {
            k_cond_out<<<(unsigned)((2 * nw + 127) / 128), 128, 0, st>>>(2 * nw, ws.kappa2, reinterpret_cast<double*>(out) + 2 * w0);
            CK(cudaGetLastError());
            c->launches++;
        } else if (call == CALL_OVERLAP) {
            CK(launch_dets(c, 0, nw, ws, st));
            shard_reduce(c, ws, st);
            mark(c, 2, st);
            CK(launch_finish_overlap(c, nw, ws, out + w0, fl, st));
            mark(c, 3, st); mark(c, 4, st); mark(c, 5, st);
        } else if (call == CALL_PROPAGATE) {
            // one phaseless-AFQMC step (propagate.cu): force bias and overlap of the walkers as they are, the field
            // matrices of all walkers as one DMMA contraction, the orbital update in place, the overlap of the new walkers
            cplx* pa_rw = const_cast<cplx*>(pa); cplx* pb_rw = const_cast<cplx*>(pb);
            CK(launch_dets(c, 1, nw, ws, st));
            shard_reduce(c, ws, st);
            mark(c, 2, st);
            CK(launch_green_rows(c, nw, ws, nullptr, st));
            CK(cudaMemsetAsync(ws.fbuf, 0, sizeof(cplx) * (size_t)nw * ng, st));
            for (int s = 0; s < 2; s++) {
                const auto& sp = c->sp[s];
                if (sp.n_r == 0) continue;
                CK(launch_fb_gemm(c, s, nw, ws, ws.fbuf, st));
            }
            CK(launch_finish_overlap(c, nw, ws, ws.ov_old, ws.fl_old, st));
            mark(c, 3, st);
            CK(launch_prop_fields(c, nw, c->prop_x + w0 * (int64_t)ng, ws.fbuf, ws.Yf, ws.expo, st));
            CK(launch_prop_vhs(c, nw, ws.Yf, ws.Aw, st));
            CK(launch_prop_orbitals(c, nw, ws.Aw, pa_rw, pb_rw, st));
            mark(c, 4, st);
            CK(cudaMemsetAsync(ws.zero_begin, 0, ws.zero_bytes, st));
            CK(launch_reference(c, N, ldN, c->dev(0), c->dev(1), nw, pa, pb, ws, false, st));
            c->launches++;
            CK(launch_dets(c, 0, nw, ws, st));
            shard_reduce(c, ws, st);
            CK(launch_finish_overlap(c, nw, ws, ws.ov_new, fl, st));
            mark(c, 5, st);
            CK(launch_prop_finish(c, nw, ws.ov_old, ws.ov_new, ws.expo, c->prop_w ? c->prop_w + w0 : nullptr,
                                  reinterpret_cast<double*>(out) + w0 * 8, ws.fl_old, fl, st));
        } else if (call == CALL_FB || call == CALL_GREENS) {
            CK(launch_dets(c, 1, nw, ws, st));
            shard_reduce(c, ws, st);
            mark(c, 2, st);
            if (call == CALL_GREENS) {
                cplx* G = out + w0 * (int64_t)2 * N * N;
                CK(cudaMemsetAsync(G, 0, sizeof(cplx) * (size_t)nw * 2 * N * N, st));
                double* keep[2] = {ws.Gp[0], ws.Gp[1]};
                ws.Gp[0] = ws.Gp[1] = nullptr;
                cudaError_t e = launch_green_rows(c, nw, ws, G, st);
                ws.Gp[0] = keep[0]; ws.Gp[1] = keep[1];
                CK(e);
                mark(c, 3, st);
                CK(launch_finish_flags(c, nw, ws, G, (int64_t)2 * N * N, fl, st));
            } else {
                CK(launch_green_rows(c, nw, ws, nullptr, st));
                cplx* fb = out + w0 * (int64_t)ng;
                CK(cudaMemsetAsync(fb, 0, sizeof(cplx) * (size_t)nw * ng, st));
                {   // the two spins' contractions only meet in the RED accumulators of fb: side by side on two streams
                    Fork ff(c, st);
                    for (int s = 0; s < 2; s++) {
                        const auto& sp = c->sp[s];
                        if (sp.n_r == 0) continue;
                        cudaError_t ge = launch_fb_gemm(c, s, nw, ws, fb, ff.stream(s));
                        if (ge != cudaSuccess) { ff.join(); CK(ge); }
                    }
                    CK(ff.join());
                }
                mark(c, 3, st);
                // msd_force_bias_overlap: the pass has W and det0 of every walker anyway (no second determinant pass)
                if (c->fb_ovlp) CK(launch_finish_overlap(c, nw, ws, c->fb_ovlp + w0, nullptr, st));
                CK(launch_finish_flags(c, nw, ws, fb, ng, fl, st));
            }
            mark(c, 4, st); mark(c, 5, st);
        } else {   // energy
            // S7: Lambda = L_sub Theta and the dense intermediates.  Fused kernel (Lambda never leaves the SM) when the shape is
            // covered, else the Lambda GEMM + dense kernel pair
            cudaError_t fe = c->no_fused ? cudaErrorNotSupported : launch_energy_fused(c, nw, ws, st);
            if (fe != cudaSuccess && fe != cudaErrorNotSupported) CK(fe);
            if (fe == cudaErrorNotSupported) {
                cudaGetLastError();
                Fork fl_(c, st);
                for (int s = 0; s < 2; s++) {
                    const auto& sp = c->sp[s];
                    if (sp.n == 0 || sp.n_r == 0) continue;
                    GemmArgs a;
                    a.A = sp.d_Lsub; a.B = ws.thetaT[s]; a.C = reinterpret_cast<double*>(ws.Lam[s]);
                    a.M = (ng + 1) * sp.n_r; a.N = (int)(2 * sp.n * nw); a.K = ldN;
                    a.lda = ldN; a.ldb = ldN; a.strideA = 0; a.strideB = 0; a.batch = 1;
                    a.zdiv = 1; a.strideC_hi = 0; a.strideC_lo = 0; a.cs_m = (int64_t)nw * sp.n; a.cs_j = 1;
                    a.accumulate = 0;
                    cudaError_t ge = launch_gemm_tn(c, a, fl_.stream(s));
                    if (ge != cudaSuccess) { fl_.join(); CK(ge); }
                    c->launches++;
                }
                CK(fl_.join());
                mark(c, 2, st);
                CK(launch_energy_dense(c, nw, ws, st));
            } else mark(c, 2, st);
            mark(c, 3, st);
            // V GEMMs: ab, aa, bb
            Fork fv_(c, st);
            for (int pr = 0; pr < 3; pr++) {
                const int s1 = (pr == 2) ? 1 : 0, s2 = (pr == 0) ? 1 : s1;
                const auto& A_ = c->sp[s1]; const auto& B_ = c->sp[s2];
                if (A_.P == 0 || B_.P == 0) continue;
                if (pr > 0 && A_.kmax < 2) continue;          // same-spin V only feeds levels >= 2
                GemmArgs a;
                a.A = reinterpret_cast<const double*>(ws.Bp[s1]); a.B = reinterpret_cast<const double*>(ws.Bp[s2]);
                a.bexpand = 1;
                a.C = reinterpret_cast<double*>(pr == 0 ? ws.Vab : ws.Vss[s1]);
                a.M = A_.P; a.N = 2 * B_.P; a.K = 2 * ng;
                a.lda = 2 * ng; a.ldb = 2 * ng;
                a.strideA = (int64_t)A_.P * 2 * ng; a.strideB = (int64_t)B_.P * 2 * ng; a.batch = (int)nw;
                a.zdiv = MSD_WT; a.strideC_hi = (int64_t)A_.P * B_.P * MSD_WT; a.strideC_lo = 1;
                a.cs_m = (int64_t)B_.P * MSD_WT; a.cs_j = MSD_WT;
                a.accumulate = 0;
                a.symmetric = (pr > 0) ? 1 : 0;     // V^{ss}[x][y] = V^{ss}[y][x]
                // 3-multiplication kernel for the well-conditioned walkers, 4-multiplication kernel for the others (both are
                // launched over the whole batch and skip the walkers of the other kind on the device: no host round trip)
                cudaError_t ge = cudaSuccess;
                if (c->no_3m || c->v3m_max_cond <= 0.0) ge = launch_gemm_tn(c, a, fv_.stream(pr));
                else {
                    a.sel = ws.kappa2; a.sel_thr = c->v3m_max_cond * c->v3m_max_cond; a.sel_hi = 0;
                    ge = launch_vgemm3m(c, a, fv_.stream(pr));
                    if (ge == cudaSuccess) { a.sel_hi = 1; c->launches++; ge = launch_gemm_tn(c, a, fv_.stream(pr)); }
                }
                if (ge != cudaSuccess) { fv_.join(); CK(ge); }
                c->launches++;
            }
            {   // F += sum_g Xt_g B^g next to the GEMMs (side stream 3)
                cudaError_t fe = launch_fx(c, nw, ws, fv_.stream(3));
                if (fe != cudaSuccess) { fv_.join(); CK(fe); }
            }
            CK(fv_.join());
            mark(c, 4, st);
            if (call == CALL_FB_ENERGY) {
                // fused call: the energy-mode dets kernels also scatter C; the force bias then comes from C and the
                // B^gamma slices that the energy path holds anyway (W6), rows of [n_chol + 3]: fb, then (E, E1, E2)
                const int64_t stride = (int64_t)ng + 3;
                CK(launch_dets(c, 3, nw, ws, st));
                shard_reduce(c, ws, st);
                mark(c, 5, st);
                CK(launch_fb_from_cb(c, nw, ws, out + w0 * stride, stride, st));
                CK(launch_finish_energy(c, nw, ws, out + w0 * stride + ng, stride, fl, st));
            } else {
                CK(launch_dets(c, 2, nw, ws, st));
                shard_reduce(c, ws, st);
                mark(c, 5, st);
                CK(launch_finish_energy(c, nw, ws, out + w0 * 3, 3, fl, st));
            }
        }
        if (c->profiling) {
            cudaEventRecord(c->ev[6], st);
            CK(cudaEventSynchronize(c->ev[6]));
            for (int i = 0; i < 6; i++) {
                float ms = 0.f;
                cudaEventElapsedTime(&ms, c->ev[i], c->ev[i + 1]);
                c->phase_ms[i] += ms;
            }
        }
    }
    return MSD_OK;
}

static int hot_call(msd_ctx* c, int call, int64_t n_w, const void* phi_a, const void* phi_b, void* out, int32_t* flags,
                    void* stream)
{
    if (!c) return MSD_EINVAL;
    if (n_w < 0 || (n_w > 0 && (!out || (c->sp[0].n > 0 && !phi_a) || (c->sp[1].n > 0 && !phi_b)))) {
        c->err = "bad argument";
        return MSD_EINVAL;
    }
    if (n_w == 0) return MSD_OK;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != c->device) { c->err = "context used on another device"; return MSD_EINVAL; }
    std::string err;
    int rc = run_chunks(c, &err, call, n_w, (const cplx*)phi_a, (const cplx*)phi_b, (cplx*)out, flags, (cudaStream_t)stream);
    if (rc != MSD_OK) { c->err = err; cudaGetLastError(); }
    return rc;
}

extern "C" int msd_overlap(msd_ctx* c, int64_t n_w, const void* phi_a, const void* phi_b, void* ovlp, int32_t* flags,
                           void* stream)
{ return hot_call(c, CALL_OVERLAP, n_w, phi_a, phi_b, ovlp, flags, stream); }

extern "C" int msd_force_bias(msd_ctx* c, int64_t n_w, const void* phi_a, const void* phi_b, void* fb, int32_t* flags,
                              void* stream)
{ return hot_call(c, CALL_FB, n_w, phi_a, phi_b, fb, flags, stream); }

extern "C" int msd_reference_cond(msd_ctx* c, int64_t n_w, const void* phi_a, const void* phi_b, double* cond, void* stream)
{ return hot_call(c, CALL_COND, n_w, phi_a, phi_b, cond, nullptr, stream); }

extern "C" int msd_force_bias_overlap(msd_ctx* c, int64_t n_w, const void* phi_a, const void* phi_b, void* fb, void* ovlp,
                                      int32_t* flags, void* stream)
{
    if (!c) return MSD_EINVAL;
    if (n_w > 0 && !ovlp) { c->err = "bad argument"; return MSD_EINVAL; }
    c->fb_ovlp = (cplx*)ovlp;
    const int rc = hot_call(c, CALL_FB, n_w, phi_a, phi_b, fb, flags, stream);
    c->fb_ovlp = nullptr;
    return rc;
}

extern "C" int msd_local_energy(msd_ctx* c, int64_t n_w, const void* phi_a, const void* phi_b, void* e, int32_t* flags,
                                void* stream)
{ return hot_call(c, CALL_ENERGY, n_w, phi_a, phi_b, e, flags, stream); }

extern "C" int msd_force_bias_energy(msd_ctx* c, int64_t n_w, const void* phi_a, const void* phi_b, void* out, int32_t* flags,
                                     void* stream)
{ return hot_call(c, CALL_FB_ENERGY, n_w, phi_a, phi_b, out, flags, stream); }

extern "C" int msd_propagator_setup(msd_ctx* c, double dt, int n_taylor, const double* h1, const double* L, void* stream)
{
    if (!c) return MSD_EINVAL;
    if (!(dt > 0.0) || n_taylor < 1 || n_taylor > 64 || !h1 || !L) { c->err = "bad argument"; return MSD_EINVAL; }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != c->device) { c->err = "context used on another device"; return MSD_EINVAL; }
    cudaError_t e = prop_setup(c, dt, n_taylor, h1, L, (cudaStream_t)stream);
    if (e != cudaSuccess) {
        c->err = std::string("propagator setup failed: ") + cudaGetErrorString(e);
        cudaGetLastError();
        return e == cudaErrorMemoryAllocation ? MSD_ENOMEM : MSD_ECUDA;
    }
    return MSD_OK;
}

extern "C" int msd_propagate(msd_ctx* c, int64_t n_w, void* phi_a, void* phi_b, const double* x, double* weights,
                             double* step_out, int32_t* flags, void* stream)
{
    if (!c) return MSD_EINVAL;
    if (c->prop_dt <= 0.0) { c->err = "msd_propagator_setup has not been called"; return MSD_EINVAL; }
    if (n_w > 0 && !x) { c->err = "bad argument"; return MSD_EINVAL; }
    c->prop_x = x; c->prop_w = weights;
    return hot_call(c, CALL_PROPAGATE, n_w, phi_a, phi_b, step_out, flags, stream);
}

extern "C" int msd_greens(msd_ctx* c, int64_t n_w, const void* phi_a, const void* phi_b, void* G, int32_t* flags,
                          void* stream)
{ return hot_call(c, CALL_GREENS, n_w, phi_a, phi_b, G, flags, stream); }

// ---------------------------------------------------------------------------------------------
// HOST-buffer variants: H2D of the walkers, the hot call, D2H of the result, all on `stream`, synchronised before
// returning.  The staging buffers belong to the context (grown on demand).
// ---------------------------------------------------------------------------------------------
static int ensure_staging(msd_ctx* c, int64_t n_w, size_t out_elems_per_walker, std::string* errp)
{
    const size_t need_a = sizeof(cplx) * (size_t)n_w * c->N * c->sp[0].n;
    const size_t need_b = sizeof(cplx) * (size_t)n_w * c->N * c->sp[1].n;
    const size_t need_o = sizeof(cplx) * (size_t)n_w * out_elems_per_walker;
    const size_t need_f = sizeof(int32_t) * (size_t)n_w;
    auto grow = [&](void** p, size_t* have, size_t need) -> cudaError_t {
        if (*have >= need && *p) return cudaSuccess;
        if (*p) { cudaError_t e = cudaDeviceSynchronize(); if (e != cudaSuccess) return e; cudaFree(*p); *p = nullptr; *have = 0; }
        cudaError_t e = cudaMalloc(p, std::max<size_t>(need, 16));
        if (e == cudaSuccess) *have = std::max<size_t>(need, 16);
        return e;
    };
    CK(grow(&c->stg_a, &c->stg_a_bytes, need_a));
    CK(grow(&c->stg_b, &c->stg_b_bytes, need_b));
    CK(grow(&c->stg_out, &c->stg_out_bytes, need_o));
    CK(grow(&c->stg_flags, &c->stg_flags_bytes, need_f));
    return MSD_OK;
}

static int hot_call_host(msd_ctx* c, int call, size_t per_walker, int64_t n_w, const void* phi_a, const void* phi_b,
                         void* out, int32_t* flags, void* stream)
{
    if (!c) return MSD_EINVAL;
    if (n_w < 0 || (n_w > 0 && (!out || (c->sp[0].n > 0 && !phi_a) || (c->sp[1].n > 0 && !phi_b)))) {
        c->err = "bad argument";
        return MSD_EINVAL;
    }
    if (n_w == 0) return MSD_OK;
    cudaStream_t st = (cudaStream_t)stream;
    std::string err;
    std::string* errp = &err;
    int rc = ensure_staging(c, n_w, per_walker, errp);
    if (rc != MSD_OK) { c->err = err; cudaGetLastError(); return rc; }
    auto body = [&]() -> int {
        const size_t ba = sizeof(cplx) * (size_t)n_w * c->N * c->sp[0].n, bb = sizeof(cplx) * (size_t)n_w * c->N * c->sp[1].n;
        if (ba) CK(cudaMemcpyAsync(c->stg_a, phi_a, ba, cudaMemcpyHostToDevice, st));
        if (bb) CK(cudaMemcpyAsync(c->stg_b, phi_b, bb, cudaMemcpyHostToDevice, st));
        int r = hot_call(c, call, n_w, c->stg_a, c->stg_b, c->stg_out, flags ? (int32_t*)c->stg_flags : nullptr, stream);
        if (r != MSD_OK) { err = c->err; return r; }
        CK(cudaMemcpyAsync(out, c->stg_out, sizeof(cplx) * (size_t)n_w * per_walker, cudaMemcpyDeviceToHost, st));
        if (flags) CK(cudaMemcpyAsync(flags, c->stg_flags, sizeof(int32_t) * (size_t)n_w, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        return MSD_OK;
    };
    rc = body();
    if (rc != MSD_OK) { c->err = err; cudaGetLastError(); }
    return rc;
}

extern "C" int msd_overlap_host(msd_ctx* c, int64_t n_w, const void* phi_a, const void* phi_b, void* ovlp, int32_t* flags,
                                void* stream)
{ return hot_call_host(c, CALL_OVERLAP, 1, n_w, phi_a, phi_b, ovlp, flags, stream); }

extern "C" int msd_force_bias_host(msd_ctx* c, int64_t n_w, const void* phi_a, const void* phi_b, void* fb, int32_t* flags,
                                   void* stream)
{ return hot_call_host(c, CALL_FB, c ? (size_t)c->n_chol : 0, n_w, phi_a, phi_b, fb, flags, stream); }

extern "C" int msd_force_bias_energy_host(msd_ctx* c, int64_t n_w, const void* phi_a, const void* phi_b, void* out,
                                          int32_t* flags, void* stream)
{ return hot_call_host(c, CALL_FB_ENERGY, c ? (size_t)c->n_chol + 3 : 0, n_w, phi_a, phi_b, out, flags, stream); }

extern "C" int msd_local_energy_host(msd_ctx* c, int64_t n_w, const void* phi_a, const void* phi_b, void* e, int32_t* flags,
                                     void* stream)
{ return hot_call_host(c, CALL_ENERGY, 3, n_w, phi_a, phi_b, e, flags, stream); }

// ---------------------------------------------------------------------------------------------
// No-allocation variant of the overlap call (include/msd.h: msd_noalloc_setup, msd_overlap_noalloc).
//
// For callers that cannot allocate in the hot loop (code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc): the per-call workspace of msd_overlap -- the zeroed per-walker accumulators C^a, C^b, W, the reference data
// Theta, g, det0 -- is carved out of ONE file-scope device array of MSD_NOALLOC_SCRATCH_BYTES instead of the context's
// cudaMalloc'ed workspace.  Every GPU that loads the library holds the array until the process exits.
//
// g_noalloc_scratch names the array in DEVICE code only (k_noalloc_clear below uses it directly).  In host code the same
// name is a host-side stand-in, not a device address: the address the kernels get comes from cudaGetSymbolAddress, taken once
// per device at set-up (msd_noalloc_setup) with that device current.
// All contexts and all calls on a device share the array and it keeps the previous call's contents: the accumulator region is
// cleared at the start of every call, and calls that overlap on the GPU (two streams, two threads, two contexts) race.
// ---------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_noalloc_scratch[MSD_NOALLOC_SCRATCH_BYTES];

static const int NOALLOC_MAX_DEVICES = 64;
static char* g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {};      // device address of g_noalloc_scratch on device d (0: not set up)
static std::mutex g_noalloc_mu;

// clears the first n16 16-byte words of the scratch array (the accumulators that must start at zero)
__global__ void k_noalloc_clear(size_t n16)
{
    uint4* p = reinterpret_cast<uint4*>(g_noalloc_scratch);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (size_t)gridDim.x * blockDim.x)
        p[i] = make_uint4(0u, 0u, 0u, 0u);
}

extern "C" int msd_noalloc_setup(msd_ctx* c, void* stream)
{
    if (!c) return MSD_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != c->device) { c->err = "context used on another device"; return MSD_EINVAL; }
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) { c->err = "device ordinal beyond the no-allocation table"; return MSD_EUNSUPPORTED; }
    if (c->shard_world > 1) { c->err = "msd_overlap_noalloc does not take determinant-sharded contexts"; return MSD_EUNSUPPORTED; }
    {
        std::lock_guard<std::mutex> lk(g_noalloc_mu);
        if (!g_noalloc_ptr[dev]) {
            char* p = nullptr;
            cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
            if (e != cudaSuccess || !p) {
                c->err = std::string("cudaGetSymbolAddress(g_noalloc_scratch): ") + cudaGetErrorString(e);
                cudaGetLastError();
                return MSD_ECUDA;
            }
            g_noalloc_ptr[dev] = p;
        }
    }
    // everything the hot call would otherwise create lazily: the context's side streams and fork/join events ...
    {
        Fork f(c, st);
        f.stream(1);
        cudaError_t e = f.join();
        if (e != cudaSuccess || f.err != cudaSuccess) { c->err = "creating the side streams failed"; cudaGetLastError(); return MSD_ECUDA; }
    }
    // (The kernels' shared-memory attributes and occupancy entries are set by func_config at their first launch:
    // cudaFuncSetAttribute and the occupancy query allocate nothing.)
    c->noalloc_ready = true;
    return MSD_OK;
}

extern "C" int msd_overlap_noalloc(msd_ctx* c, int64_t n_w, const void* phi_a, const void* phi_b, void* ovlp, int32_t* flags,
                                   void* stream)
{
    if (!c) return MSD_EINVAL;
    if (n_w < 0 || (n_w > 0 && (!ovlp || (c->sp[0].n > 0 && !phi_a) || (c->sp[1].n > 0 && !phi_b)))) {
        c->err = "bad argument";
        return MSD_EINVAL;
    }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != c->device) { c->err = "context used on another device"; return MSD_EINVAL; }
    if (!c->noalloc_ready || dev < 0 || dev >= NOALLOC_MAX_DEVICES || !g_noalloc_ptr[dev]) {
        c->err = "msd_overlap_noalloc: call msd_noalloc_setup(ctx) first (once per context, outside the no-allocation region)";
        return MSD_EINVAL;
    }
    if (n_w == 0) return MSD_OK;
    cudaStream_t st = (cudaStream_t)stream;
    // layout of the overlap workspace (level 1) for the whole batch: no chunking here, a batch that does not fit is refused
    const int64_t wc = (n_w + MSD_WT - 1) / MSD_WT * MSD_WT;
    Workspace ws;
    const size_t need = carve(c, ws, nullptr, wc, 1);
    if (need > (size_t)MSD_NOALLOC_SCRATCH_BYTES) {
        char msg[256];
        snprintf(msg, sizeof msg, "msd_overlap_noalloc: n_w = %lld needs %zu bytes of scratch, the library holds "
                 "MSD_NOALLOC_SCRATCH_BYTES = %d; split the batch or use msd_overlap", (long long)n_w, need, MSD_NOALLOC_SCRATCH_BYTES);
        c->err = msg;
        return MSD_ENOMEM;
    }
    char* base = g_noalloc_ptr[dev];                // a device address (cudaGetSymbolAddress), never &g_noalloc_scratch
    carve(c, ws, base, wc, 1);
    ws.wc = wc; ws.want = wc; ws.level = 1; ws.base = base; ws.bytes = MSD_NOALLOC_SCRATCH_BYTES;
    const int N = c->N, ldN = N + (N & 1);
    std::string err;
    auto run = [&]() -> int {
        std::string* errp = &err;
        // the zero region is the first zero_bytes of the array (carve puts it first; a multiple of 256 bytes)
        if (ws.zero_begin != base) return fail(errp, MSD_ECUDA, "unexpected workspace layout");
        const size_t n16 = ws.zero_bytes / 16;
        const unsigned blocks = (unsigned)std::min<size_t>((n16 + 255) / 256, (size_t)c->n_sm * 8);
        k_noalloc_clear<<<blocks ? blocks : 1, 256, 0, st>>>(n16);
        CK(cudaGetLastError());
        c->launches++;
        CK(launch_reference(c, N, ldN, c->dev(0), c->dev(1), n_w, (const cplx*)phi_a, (const cplx*)phi_b, ws, false, st));
        c->launches++;
        CK(launch_dets(c, 0, n_w, ws, st));
        CK(launch_finish_overlap(c, n_w, ws, (cplx*)ovlp, flags, st));
        return MSD_OK;
    };
    const int rc = run();
    if (rc != MSD_OK) { c->err = err; cudaGetLastError(); }
    return rc;
}

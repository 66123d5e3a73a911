// Bench-side peak probes (libmsd_probes.so): roofline DENOMINATORS measured on the box bench.py runs on.
// Not part of the product ABI (include/msd.h) and not linked into libmsd_b200.so; only bench.py loads this.
//   msd_probe_fp64_tflops : register-resident DMMA m8n8k4 (or DFMA) loop -> FP64 peak.  MEASURED_PEAKS.json has no FP64
//                           entry and the profiling guide lists no FP64 nominal for sm_100a.
//   msd_probe_l2_gather_gbs : the access pattern of the energy-mode determinant kernels -- every 8 lanes read one random
//                           128-byte line (16 B per lane) of an L2-resident buffer, several independent loads in
//                           flight per lane -> L2 -> SM gather bandwidth.
#include <cuda_runtime.h>
#include <stdint.h>

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

__global__ void k_probe_dmma(double* out, int iters)
{
    double d[8][2];
    for (int j = 0; j < 8; j++) { d[j][0] = 0.0; d[j][1] = 0.0; }
    double a = threadIdx.x * 1e-3, b = 1e-3;
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int j = 0; j < 8; j++) dmma884(d[j][0], d[j][1], a, b);
    }
    double s = 0.0;
    for (int j = 0; j < 8; j++) s += d[j][0] + d[j][1];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void k_probe_dfma(double* out, int iters)
{
    double a[8];
    for (int j = 0; j < 8; j++) a[j] = threadIdx.x * 1e-9 + j;
    const double b = 1.0000001, c = 1e-9;
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int j = 0; j < 8; j++) a[j] = fma(a[j], b, c);
    }
    double s = 0.0;
    for (int j = 0; j < 8; j++) s += a[j];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

extern "C" double msd_probe_fp64_tflops(int use_dmma, double ms_target, void* stream)
{
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1.0;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    const int thr = 512, blocks = nsm * 2;
    double* out = nullptr;
    if (cudaMalloc(&out, sizeof(double) * thr * blocks) != cudaSuccess) return -1.0;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    int iters = 20000;
    double best = 0.0;
    for (int rep = 0; rep < 3; rep++) {
        cudaEventRecord(e0, st);
        if (use_dmma) k_probe_dmma<<<blocks, thr, 0, st>>>(out, iters);
        else k_probe_dfma<<<blocks, thr, 0, st>>>(out, iters);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { best = -1.0; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        double fl = use_dmma ? 2.0 * 8 * 8 * 4 * 8 * (double)iters * blocks * thr / 32.0
                             : 2.0 * 8 * (double)iters * blocks * thr;
        double tf = fl / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best) best = tf;
        if (rep == 0 && ms > 0.f && ms_target > 0.0) {
            double scale = ms_target / ms;
            if (scale > 200.0) scale = 200.0;
            if (scale > 1.0) iters = (int)(iters * scale);
        }
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    return best;
}

// lane (q = lane / 8, j = lane % 8) reads element j of line `idx` -- 8 lanes cover one 128-byte line; UNR independent
// line indices per iteration from a per-group LCG
template <int UNR>
__global__ void __launch_bounds__(256) k_probe_l2_gather(const double2* __restrict__ buf, unsigned nlines_mask, int iters,
                                                         double* out)
{
    const int j = threadIdx.x & 7;
    unsigned state = (blockIdx.x * 256u + (threadIdx.x >> 3)) * 2654435761u + 12345u;
    double2 acc = make_double2(0.0, 0.0);
    for (int it = 0; it < iters; it++) {
        double2 v[UNR];
#pragma unroll
        for (int u = 0; u < UNR; u++) {
            state = state * 1664525u + 1013904223u;
            const unsigned line = (state >> 8) & nlines_mask;
            v[u] = __ldg(buf + (size_t)line * 8 + j);
        }
#pragma unroll
        for (int u = 0; u < UNR; u++) { acc.x += v[u].x; acc.y += v[u].y; }
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc.x + acc.y;
}

// buffer of `mbytes` MB (power of two; stays in the 126 MB L2 when <= 64); returns GB/s of gathered bytes
extern "C" double msd_probe_l2_gather_gbs(int mbytes, double ms_target, void* stream)
{
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1.0;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    size_t bytes = (size_t)mbytes << 20;
    unsigned nlines = (unsigned)(bytes / 128);
    if (nlines == 0 || (nlines & (nlines - 1))) return -1.0;
    double2* buf = nullptr; double* out = nullptr;
    const int thr = 256, blocks = nsm * 8;
    if (cudaMalloc(&buf, bytes) != cudaSuccess) return -1.0;
    if (cudaMalloc(&out, sizeof(double) * thr * blocks) != cudaSuccess) { cudaFree(buf); return -1.0; }
    cudaMemsetAsync(buf, 0, bytes, st);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    int iters = 200;
    double best = 0.0;
    constexpr int UNR = 8;
    for (int rep = 0; rep < 4; rep++) {
        cudaEventRecord(e0, st);
        k_probe_l2_gather<UNR><<<blocks, thr, 0, st>>>(buf, nlines - 1, iters, out);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { best = -1.0; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        double gbs = 16.0 * UNR * (double)iters * blocks * thr / (ms * 1e-3) / 1e9;
        if (rep > 0 && gbs > best) best = gbs;
        if (rep == 0 && ms > 0.f && ms_target > 0.0) {
            double scale = ms_target / ms;
            if (scale > 500.0) scale = 500.0;
            if (scale > 1.0) iters = (int)(iters * scale);
        }
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(buf); cudaFree(out);
    return best;
}

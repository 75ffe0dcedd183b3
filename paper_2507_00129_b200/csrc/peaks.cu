// peaks.cu -- liblya_peaks.so (include/lya_peaks.h): microbenchmarks of the units that bound the
// pair loops (fp64 pipe issue rate, shared-memory atomics, L2 fp64 reductions).  They give the
// MEASURED roofline denominators quoted in DESIGN.md / bench.py.  Built as its own library: the
// product library liblya.so does not contain them.
#include <cuda_runtime.h>
#include "../../include/lya_peaks.h"

namespace {

constexpr int PK_THREADS = 256;

template <bool FMA>
__global__ void k_peak_fp64(double *out, int iters, double b, double c)
{
    double a0 = threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    for (int i = 0; i < iters; ++i) {
        if (FMA) {
            a0 = fma(a0, b, c); a1 = fma(a1, b, c); a2 = fma(a2, b, c); a3 = fma(a3, b, c);
            a4 = fma(a4, b, c); a5 = fma(a5, b, c); a6 = fma(a6, b, c); a7 = fma(a7, b, c);
        } else {
            a0 = __dadd_rn(a0, c); a1 = __dadd_rn(a1, c); a2 = __dadd_rn(a2, c); a3 = __dadd_rn(a3, c);
            a4 = __dadd_rn(a4, c); a5 = __dadd_rn(a5, c); a6 = __dadd_rn(a6, c); a7 = __dadd_rn(a7, c);
        }
    }
    double r = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (r == 123.456) out[0] = r;       // never true; keeps the chain alive
}

template <bool F64>
__global__ void k_peak_smem(unsigned long long *out, int iters, int nbins)
{
    extern __shared__ __align__(16) unsigned char raw[];
    double *hd = (double *)raw;
    unsigned *hu = (unsigned *)raw;
    for (int k = threadIdx.x; k < nbins; k += blockDim.x) { if (F64) hd[k] = 0.0; else hu[k] = 0u; }
    __syncthreads();
    unsigned x = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 12345u;
    for (int i = 0; i < iters; ++i) {
        x = x * 1664525u + 1013904223u;
        unsigned bin = (unsigned)(((unsigned long long)(x >> 8) * (unsigned)nbins) >> 24);
        if (F64) atomicAdd(&hd[bin], 1.0); else atomicAdd(&hu[bin], 1u);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long t = F64 ? (unsigned long long)hd[0] : hu[0];
        if (t == 0xffffffffffffull) out[0] = t;
    }
}

__global__ void k_peak_red(double *mat, int nb, int iters)
{
    const int lane = threadIdx.x & 31;
    unsigned x = ((blockIdx.x * blockDim.x + threadIdx.x) >> 5) * 2654435761u + 777u;
    for (int i = 0; i < iters; ++i) {
        x = x * 1664525u + 1013904223u;
        unsigned row = (unsigned)(((unsigned long long)(x >> 8) * (unsigned)nb) >> 24);
        x = x * 1664525u + 1013904223u;
        unsigned col = (unsigned)(((unsigned long long)(x >> 8) * (unsigned)(nb - 32)) >> 24);
        atomicAdd(&mat[(size_t)row * nb + col + lane], 1.0);
    }
}

// every lane its own random element of an n-element array (the access pattern of k_xi3: 32 sectors per instruction)
__global__ void k_peak_red_scatter(double *mat, unsigned n, int iters)
{
    unsigned x = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 4242u;
    for (int i = 0; i < iters; ++i) {
        x = x * 1664525u + 1013904223u;
        atomicAdd(&mat[(unsigned)(((unsigned long long)x * n) >> 32)], 1.0);
    }
}

}  // namespace

extern "C" int lya_measure_peak(int device, lya_peak_kind kind, double *rate)
{
    if (!rate) return (int)cudaErrorInvalidValue;
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return (int)e;
    cudaDeviceProp prop;
    if ((e = cudaGetDeviceProperties(&prop, device)) != cudaSuccess) return (int)e;
    const int grid = prop.multiProcessorCount * 4;
    cudaEvent_t ev0, ev1;
    if ((e = cudaEventCreate(&ev0)) != cudaSuccess) return (int)e;
    if ((e = cudaEventCreate(&ev1)) != cudaSuccess) { cudaEventDestroy(ev0); return (int)e; }
    cudaStream_t s = 0;
    double ops = 0.0;
    float ms = 0.f;
    double *buf = NULL;
    const int nb = 2500;
    auto done = [&](cudaError_t err) { cudaFree(buf); cudaEventDestroy(ev0); cudaEventDestroy(ev1); return (int)err; };
    if ((e = cudaMalloc(&buf, sizeof(double) * (size_t)nb * nb)) != cudaSuccess) return done(e);
    cudaMemsetAsync(buf, 0, sizeof(double) * (size_t)nb * nb, s);
    for (int rep = 0; rep < 2; ++rep) {          // rep 0 = warm-up
        cudaEventRecord(ev0, s);
        switch (kind) {
        case LYA_PEAK_FP64_FMA: {
            int iters = 1 << 14;
            k_peak_fp64<true><<<grid, PK_THREADS, 0, s>>>(buf, iters, 1.0000001, 1e-9);
            ops = (double)grid * PK_THREADS * 8.0 * iters;
            break; }
        case LYA_PEAK_FP64_ADD: {
            int iters = 1 << 14;
            k_peak_fp64<false><<<grid, PK_THREADS, 0, s>>>(buf, iters, 1.0000001, 1e-9);
            ops = (double)grid * PK_THREADS * 8.0 * iters;
            break; }
        case LYA_PEAK_SMEM_CAS64: {
            int iters = 1 << 12;
            k_peak_smem<true><<<grid, PK_THREADS, nb * 8, s>>>((unsigned long long *)buf, iters, nb);
            ops = (double)grid * PK_THREADS * iters;
            break; }
        case LYA_PEAK_SMEM_ADD32: {
            int iters = 1 << 12;
            k_peak_smem<false><<<grid, PK_THREADS, nb * 8, s>>>((unsigned long long *)buf, iters, nb);
            ops = (double)grid * PK_THREADS * iters;
            break; }
        case LYA_PEAK_L2_RED64: {
            int iters = 1 << 10;
            k_peak_red<<<grid, PK_THREADS, 0, s>>>(buf, nb, iters);
            ops = (double)grid * PK_THREADS * iters;
            break; }
        case LYA_PEAK_L2_RED64_SCATTER: {
            int iters = 1 << 10;
            k_peak_red_scatter<<<grid, PK_THREADS, 0, s>>>(buf, 2400000u, iters);      // 19 MB: three 800,000-bin accumulators
            ops = (double)grid * PK_THREADS * iters;
            break; }
        default:
            return done(cudaErrorInvalidValue);
        }
        cudaEventRecord(ev1, s);
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) return done(e);
        cudaEventElapsedTime(&ms, ev0, ev1);
    }
    *rate = ops / ((double)ms * 1e-3);
    return done(cudaSuccess);
}

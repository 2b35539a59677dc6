// bse_selftest_peak: the microbenchmarks behind every roofline denominator this repository quotes (DESIGN.md section 5,
// bench.py --peaks).  MEASURED_PEAKS.json holds an HBM copy figure and a bf16 GEMM figure, nothing for FP64: the FP64
// tensor (DMMA.8x8x4) and plain DFMA rates, the read-only bulk-copy stream the apply kernels are built on and the
// red.global.add.f64 rate are measured here, by kernels that do nothing else, timed with CUDA events on the caller's stream.
#include <algorithm>

#include "bse_common.cuh"
#include "bse_internal.h"

namespace bse {

// ---- FP64 tensor pipe: CHAINS independent accumulator chains per warp, nothing but DMMAs.
template <int CHAINS>
__global__ void __launch_bounds__(1024, 1) peak_dmma_kernel(double *out, int iters, double a0, double b0)
{
    double c[CHAINS][2];
#pragma unroll
    for (int q = 0; q < CHAINS; ++q) c[q][0] = c[q][1] = 0.0;
    const double a = a0 + threadIdx.x * 1e-9, b = b0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int q = 0; q < CHAINS; ++q) dmma(c[q], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < CHAINS; ++q) s += c[q][0] + c[q][1];
    if (s == 12345.678) out[0] = s;                       // never true: keeps the chains alive
}

// ---- FP64 tensor pipe shared with plain FP64 adds, the instruction mix of the three-product apply role: per group of
// 12 DMMAs (4 fragments x 3 products) 4 DADDs that each feed one DMMA operand (+ 4 that renew the operands).
__global__ void __launch_bounds__(1024, 1) peak_dmma_dadd_kernel(double *out, int iters, double a0, double b0)
{
    double c[12][2];
#pragma unroll
    for (int q = 0; q < 12; ++q) c[q][0] = c[q][1] = 0.0;
    double ar[4], ai[4];
#pragma unroll
    for (int f = 0; f < 4; ++f) { ar[f] = a0 + threadIdx.x * 1e-9 + f; ai[f] = a0 * 0.5 + f; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int f = 0; f < 4; ++f) {
            double as;
            asm volatile("add.f64 %0, %1, %2;" : "=d"(as) : "d"(ar[f]), "d"(ai[f]));
            dmma(c[3 * f], ar[f], b0);
            dmma(c[3 * f + 1], ai[f], b0);
            dmma(c[3 * f + 2], as, b0);
        }
#pragma unroll
        for (int f = 0; f < 4; ++f) ar[f] += 1e-12;
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < 12; ++q) s += c[q][0] + c[q][1];
    if (s == 12345.678) out[0] = s;
}

// ---- plain FP64 pipe: 8 independent DFMA chains per thread.
__global__ void __launch_bounds__(1024, 1) peak_dfma_kernel(double *out, int iters, double a, double b)
{
    double c[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) c[q] = threadIdx.x * 1e-9 + q;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int q = 0; q < 8; ++q) c[q] = fma(c[q], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < 8; ++q) s += c[q];
    if (s == 12345.678) out[0] = s;
}

// ---- read-only HBM stream through the bulk-copy engine: one producer lane per CTA (one CTA per SM) fills a ring of
// `stages` buffers of `chunk` bytes, one consumer warp releases them (optionally after reading every byte back from
// shared memory): the data path of the apply kernels without their arithmetic.
__global__ void __launch_bounds__(64, 1) peak_bulk_read_kernel(const char *src, int64_t n_chunks, int chunk, int stages,
                                                               int read_back, double *out)
{
    extern __shared__ __align__(1024) char smem[];
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + (size_t)stages * chunk), *empty = full + stages;
    if (threadIdx.x == 0) {
        for (int s = 0; s < stages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
        fence_barrier_init();
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int st = 0;
    uint32_t ph = 0;
    if (warp == 1) {
        if (lane == 0) {
            const uint64_t pol = l2_policy_evict_first();
            for (int64_t c = blockIdx.x; c < n_chunks; c += gridDim.x) {
                mbar_wait(&empty[st], ph ^ 1);
                mbar_expect_tx(&full[st], (uint32_t)chunk);
                bulk_g2s_hint(smem + (size_t)st * chunk, src + c * (int64_t)chunk, (uint32_t)chunk, &full[st], pol);
                if (++st == stages) { st = 0; ph ^= 1; }
            }
        }
        return;
    }
    double acc = 0.0;
    for (int64_t c = blockIdx.x; c < n_chunks; c += gridDim.x) {
        mbar_wait(&full[st], ph);
        if (read_back) {
            const double2 *p = reinterpret_cast<const double2 *>(smem + (size_t)st * chunk);
            for (int i = lane; i < chunk / 16; i += 32) { double2 v = p[i]; acc += v.x + v.y; }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[st]);
        if (++st == stages) { st = 0; ph ^= 1; }
    }
    if (acc == 12345.678) out[0] = acc;
}

// ---- red.global.add.f64 scattered over a buffer of `span` doubles (L2-resident for small spans), as the Y flushes are
__global__ void __launch_bounds__(256) peak_red_kernel(double *buf, int64_t span, int iters)
{
    const int64_t tid = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    for (int it = 0; it < iters; ++it) red_add(buf + (tid * 9 + (int64_t)it * 1031) % span, 1.0);
}

template <int CHAINS> static void launch_dmma(int grid, int threads, cudaStream_t s, double *out, int iters)
{
    peak_dmma_kernel<CHAINS><<<grid, threads, 0, s>>>(out, iters, 1.0, 1e-9);
}

// one launch of probe `what`; returns the work done (flops, bytes or atomics), 0 on invalid arguments
static double peak_launch(int what, int p1, int p2, void *dBuf, int64_t buf_bytes, cudaStream_t s, int sms, double *sink)
{
    if (what == BSE_PEAK_DMMA) {
        const int warps = std::min(std::max(p1 > 0 ? p1 : 8, 1), 32), chains = p2 != 0 ? p2 : 8;
        const int iters = 200000 / (chains > 0 ? chains : 12);
        switch (chains) {
            case -1: peak_dmma_dadd_kernel<<<sms, warps * 32, 0, s>>>(sink, iters, 1.0, 1e-9); break;
            case 1: launch_dmma<1>(sms, warps * 32, s, sink, iters); break;
            case 2: launch_dmma<2>(sms, warps * 32, s, sink, iters); break;
            case 4: launch_dmma<4>(sms, warps * 32, s, sink, iters); break;
            case 8: launch_dmma<8>(sms, warps * 32, s, sink, iters); break;
            case 12: launch_dmma<12>(sms, warps * 32, s, sink, iters); break;
            default: return 0.0;
        }
        return 2.0 * 256.0 * (double)iters * (chains > 0 ? chains : 12) * warps * sms;
    }
    if (what == BSE_PEAK_DFMA) {
        const int warps = std::min(std::max(p1 > 0 ? p1 : 32, 1), 32), iters = 100000;
        peak_dfma_kernel<<<sms, warps * 32, 0, s>>>(sink, iters, 1.0000001, 1e-9);
        return 2.0 * 8.0 * iters * warps * 32.0 * sms;
    }
    if (what == BSE_PEAK_BULK_READ || what == BSE_PEAK_BULK_READ_SMEM) {
        const int chunk = p1 > 0 ? p1 : 65536, stages = p2 > 0 ? p2 : 3;
        if (!dBuf || chunk % 16 || (size_t)chunk * stages > 220 * 1024 || buf_bytes < chunk) return 0.0;
        const int64_t n_chunks = buf_bytes / chunk;
        const int smem = chunk * stages + 16 * stages + 64;
        if (cudaFuncSetAttribute(peak_bulk_read_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return 0.0;
        peak_bulk_read_kernel<<<sms, 64, smem, s>>>((const char *)dBuf, n_chunks, chunk, stages, what == BSE_PEAK_BULK_READ_SMEM, sink);
        return (double)n_chunks * chunk;
    }
    if (!dBuf || buf_bytes < 8) return 0.0;
    const int iters = 2000, grid = sms * 8;
    peak_red_kernel<<<grid, 256, 0, s>>>((double *)dBuf, buf_bytes / 8, iters);
    return (double)iters * grid * 256.0;
}

}  // namespace bse

using namespace bse;

extern "C" bse_status_t bse_selftest_peak(int32_t what, int32_t p1, int32_t p2, void *dBuf, int64_t buf_bytes, void *stream,
                                          double *result, double *ms_out)
{
    if (!result || what < 0 || what > BSE_PEAK_RED) return BSE_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    BSE_CUDA(cudaGetDevice(&dev));
    BSE_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    cudaEvent_t e0, e1;
    BSE_CUDA(cudaEventCreate(&e0));
    BSE_CUDA(cudaEventCreate(&e1));
    double *sink = nullptr;
    BSE_CUDA(cudaMalloc(&sink, 64));
    bse_status_t st = BSE_OK;
    double work = peak_launch(what, p1, p2, dBuf, buf_bytes, s, sms, sink);          // warm-up
    float ms = 0.f;
    if (work <= 0.0) st = BSE_ERR_INVALID_ARG;
    else {
        cudaEventRecord(e0, s);
        work = peak_launch(what, p1, p2, dBuf, buf_bytes, s, sms, sink);
        cudaEventRecord(e1, s);
        count_launch(2);
        if (cudaStreamSynchronize(s) != cudaSuccess || cudaGetLastError() != cudaSuccess ||
            cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess)
            st = BSE_ERR_CUDA;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    if (st) return st;
    if (ms_out) *ms_out = ms;
    // TFLOP/s for the arithmetic probes, GB/s for the stream, G atomics/s for the reductions
    *result = (what <= BSE_PEAK_DFMA) ? work / (ms * 1e-3) / 1e12 : work / (ms * 1e-3) / 1e9;
    return BSE_OK;
}

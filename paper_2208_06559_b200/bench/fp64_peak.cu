// fp64_peak.cu -- FP64 issue-rate microbenchmark on the current device: plain DFMA and the FP64 tensor-core
// instruction the Cholesky kernels use (mma.sync m8n8k4 f64 = SASS DMMA.8x8x4; the m16n8k* f64 shapes lower to the
// same instruction on sm_100a).  Register-resident operands, no memory traffic: the ceiling of the FP64 pipes at the
// clock the GPU holds under this load.  Built as a small shared library (libbd_peak.so) so that bench.py can measure
// the roofline denominator inside the same process and run as the numbers it divides (MEASURED_PEAKS.json carries no
// FP64 entry).  Not part of libbd.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

template <int ILP>
__global__ void k_peak_dfma(double* out, int iters, double a, double b)
{
    double acc[ILP];
#pragma unroll
    for (int i = 0; i < ILP; i++) acc[i] = threadIdx.x * 1e-3 + i;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < ILP; i++) acc[i] = fma(acc[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < ILP; i++) s += acc[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <int ILP>
__global__ void k_peak_dmma884(double* out, int iters, double a, double b)
{
    double c[ILP][2];
#pragma unroll
    for (int i = 0; i < ILP; i++) { c[i][0] = threadIdx.x; c[i][1] = i; }
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < ILP; i++)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1])
                         : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < ILP; i++) s += c[i][0] + c[i][1];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace

// kind 0: DFMA (2 flop per lane and instruction), kind 1: DMMA m8n8k4 (512 flop per warp instruction).
// warps_per_sm resident warps on every SM, `iters` x 8 independent instructions per thread, best of `reps` timed
// launches after one warm-up, CUDA events on `stream`.  Returns 0 and writes TFLOP/s and the best milliseconds.
extern "C" int bdpeak_fp64(int kind, int warps_per_sm, int iters, int reps, void* stream, double* tflops, double* ms_best)
{
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1;
    if (warps_per_sm < 1 || warps_per_sm > 32 || iters < 1 || reps < 1 || (kind != 0 && kind != 1)) return -2;
    const int threads = warps_per_sm * 32;
    const int blocks = sms;
    double* out = nullptr;
    if (cudaMalloc(&out, sizeof(double) * (size_t)blocks * threads) != cudaSuccess) return -1;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    float best = 1e30f;
    for (int r = 0; r <= reps; ++r) {
        cudaEventRecord(e0, st);
        if (kind == 0) k_peak_dfma<8><<<blocks, threads, 0, st>>>(out, iters, 1.0000001, 1e-9);
        else k_peak_dmma884<8><<<blocks, threads, 0, st>>>(out, iters, 1.0000001, 1e-9);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(out); return -1; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    const double per_thread = (kind == 0) ? 2.0 * 8.0 * iters : 512.0 * 8.0 * iters / 32.0;
    *tflops = per_thread * (double)blocks * threads / ((double)best * 1e-3) / 1e12;
    *ms_best = best;
    return 0;
}

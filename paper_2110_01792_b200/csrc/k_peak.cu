// k_peak.cu -- fp64 pipe throughput probe: the roofline denominator for the ALU-bound stage
// kernels.  Every thread advances 8 independent chains; with -fmad=false
// `x * a + b` is one DMUL and one DADD (the instruction mix of the stage kernels), kind 1 uses
// __fma_rn (one DFMA).  Reports warp-level fp64 instructions x 32 lanes per second.
#include "qk_internal.h"

namespace qk {

template <int KIND>
__global__ void __launch_bounds__(256) fp64_probe_kernel(double *out, int iters, double a, double b)
{
    double x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = 1.0 + 1e-3 * (threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (KIND == 0) x[i] = x[i] * a + b;
                else           x[i] = __fma_rn(x[i], a, b);
            }
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    if (s == 123.456) out[0] = s;   // keep the chains alive
}

}  // namespace qk

extern "C" int qk_fp64_probe(int kind, int iters, void *cuda_stream, double *lane_ops_per_s)
{
    using namespace qk;
    if (!lane_ops_per_s || iters < 1 || (kind != 0 && kind != 1)) return QK_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double *d = nullptr;
    if (cudaMalloc(&d, 8) != cudaSuccess) return QK_ENOMEM;
    const int blocks = 148 * 8, threads = 256;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {     // rep 0 is the warm-up
        cudaEventRecord(e0, st);
        if (kind == 0) fp64_probe_kernel<0><<<blocks, threads, 0, st>>>(d, iters, 0.999999, 1e-6);
        else           fp64_probe_kernel<1><<<blocks, threads, 0, st>>>(d, iters, 0.999999, 1e-6);
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d);
    if (cudaGetLastError() != cudaSuccess) return QK_ECUDA;
    const double instr_per_thread = (double)iters * 4 * 8 * (kind == 0 ? 2 : 1);
    *lane_ops_per_s = instr_per_thread * blocks * threads / (best * 1e-3);
    return QK_OK;
}

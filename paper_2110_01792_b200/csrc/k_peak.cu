// k_peak.cu -- fp64 pipe throughput probe: the roofline denominator for the ALU-bound stage
// kernels.  Every thread advances 8 independent chains; with -fmad=false
// `x * a + b` is one DMUL and one DADD (the instruction mix of the stage kernels), kind 1 uses
// __fma_rn (one DFMA).  Reports warp-level fp64 instructions x 32 lanes per second.
#include "qk_internal.h"
#include "qk_fastmath.cuh"

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

// ---- self-test of the branch-free division / square root (qk_fastmath.cuh) ---------------------------------
namespace qk {

__device__ __forceinline__ unsigned long long mix64(unsigned long long z)     // splitmix64 finaliser
{
    z += 0x9e3779b97f4a7c15ull;
    z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ull;
    z = (z ^ (z >> 27)) * 0x94d049bb133111ebull;
    return z ^ (z >> 31);
}

// operand with random sign and mantissa; exponent uniform over `span` binades centred on 1 (span = 2046
// covers every normal double), and 1 in 64 operands is an exact zero, subnormal, infinity or NaN
__device__ __forceinline__ double random_operand(unsigned long long bits, int span)
{
    const unsigned long long mant = bits & 0x000fffffffffffffull;
    const unsigned long long sign = bits & 0x8000000000000000ull;
    const int pick = (int)((bits >> 52) & 0x7ff);
    if ((pick & 63) == 0) {
        const int kind = (pick >> 6) & 3;
        if (kind == 0) return __longlong_as_double((long long)sign);                                  // +-0
        if (kind == 1) return __longlong_as_double((long long)(sign | mant));                         // subnormal
        if (kind == 2) return __longlong_as_double((long long)(sign | 0x7ff0000000000000ull));        // inf
        return __longlong_as_double((long long)(0x7ff8000000000000ull | mant));                       // NaN
    }
    const unsigned long long expo = (unsigned long long)(1024 - span / 2 + pick % span);
    return __longlong_as_double((long long)(sign | (expo << 52) | mant));
}

__global__ void __launch_bounds__(256) divsqrt_selftest_kernel(long long n, unsigned long long seed, int span,
                                                               unsigned long long *out)
{
    unsigned long long acc_div = 0, bad_div = 0, acc_sqrt = 0, bad_sqrt = 0;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        const double x = random_operand(mix64(seed + 2ull * (unsigned long long)t), span);
        const double y = random_operand(mix64(seed + 2ull * (unsigned long long)t + 1ull), span);
        unsigned risk = 0;
        const double q = fdiv(x, y, risk);
        if (!risk) {
            ++acc_div;
            const double ref = x / y;
            if (__double_as_longlong(q) != __double_as_longlong(ref)) ++bad_div;
            // the variant without the range test (operands proved in range by an operand window) is the same chain
            else if (__double_as_longlong(fdiv_inrange(x, y)) != __double_as_longlong(ref)) ++bad_div;
        }
        risk = 0;
        const double ax = fabs(x);
        const double s = fsqrt(ax, risk);
        if (!risk) {
            ++acc_sqrt;
            if (__double_as_longlong(s) != __double_as_longlong(sqrt(ax))) ++bad_sqrt;
            else if (ax > 0.0 && __double_as_longlong(fsqrt_inrange(ax)) != __double_as_longlong(s)) ++bad_sqrt;
        }
    }
    atomicAdd(&out[0], acc_div); atomicAdd(&out[1], bad_div);
    atomicAdd(&out[2], acc_sqrt); atomicAdd(&out[3], bad_sqrt);
}

}  // namespace qk

extern "C" int qk_selftest_divsqrt(long long n, unsigned long long seed, int exponent_span, void *cuda_stream,
                                   long long *out4)
{
    using namespace qk;
    if (!out4 || n < 1 || exponent_span < 1 || exponent_span > 2046) return QK_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    unsigned long long *d = nullptr;
    if (cudaMalloc(&d, 32) != cudaSuccess) return QK_ENOMEM;
    cudaMemsetAsync(d, 0, 32, st);
    divsqrt_selftest_kernel<<<148 * 8, 256, 0, st>>>(n, seed, exponent_span, d);
    unsigned long long h[4];
    const bool ok = cudaMemcpyAsync(h, d, 32, cudaMemcpyDeviceToHost, st) == cudaSuccess &&
                    cudaStreamSynchronize(st) == cudaSuccess;
    cudaFree(d);
    if (!ok) { cudaGetLastError(); return QK_ECUDA; }
    for (int i = 0; i < 4; ++i) out4[i] = (long long)h[i];
    return QK_OK;
}

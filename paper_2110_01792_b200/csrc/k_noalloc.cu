// k_noalloc.cu -- qk_cfl_dt_noalloc: the eq 21 timestep of a dense hydro state WITHOUT any
// allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses
// that forbid it).  It is a variant of the CFL reduction of k_cfl.cu: that kernel accumulates into a counter block
// carved from the context's storage (qk_init / qk_bind_storage allocate it); this one needs no context and keeps its
// reduction scratch -- one partial maximum per CTA plus a bad-cell counter -- in a file-scope device array of fixed
// size, which every GPU that loads libqk.so holds until the process exits (QK_NOALLOC_SCRATCH_BYTES = 128.25 KiB).
//
//   pass 1  cfl_partial_kernel : CTA b takes the cells [1024 b, 1024 b + 1024), cons -> prim, |v| + c_s (the same
//                                operations in the same order as cfl_max_speed_kernel), block max -> part[b]; cells
//                                with rho <= 0 or P <= 0 are counted into `bad` by one atomicAdd per CTA
//   pass 2  cfl_finish_kernel  : one CTA reduces part[0 .. nblocks) and writes dt = CFL dx / max (NaN if bad != 0)
//
// A maximum does not depend on the order it is taken in, so dt equals qk_cfl_dt's double bit for bit (for c_hat = 0:
// this entry point has no radiation limit).
//
// The scratch is shared by every call in the process and keeps the last call's contents: `bad` is cleared at the
// start of every call (cudaMemsetAsync on the stream: not an allocation), every part[b] a call reads it has written
// itself.  Calls that overlap on the GPU (different streams, or several host threads) race on it: serialise them.
//
// The array's name is a host-side stand-in in host code, not a device address: the address the kernels get comes
// from cudaGetSymbolAddress, resolved once per device with that device current (noalloc_scratch below).
#include <mutex>

#include "qk_internal.h"
#include "qk_math.cuh"

namespace qk {

constexpr int NA_THREADS = 256, NA_CELLS_PER_THREAD = 4;
constexpr int NA_CELLS_PER_BLOCK = NA_THREADS * NA_CELLS_PER_THREAD;            // 1024
constexpr long long NA_MAX_BLOCKS = QK_NOALLOC_MAX_CELLS / NA_CELLS_PER_BLOCK;  // 16384
constexpr int NA_HEADER = 32;                                                   // 256 B: word 0 = bad-cell counter
static_assert((NA_HEADER + NA_MAX_BLOCKS) * 8 == QK_NOALLOC_SCRATCH_BYTES, "qk.h states the scratch size");

// [0] bad-cell counter, [1..31] unused, [32 + b] bit pattern of the partial maximum of CTA b
static __device__ __align__(256) unsigned long long qk_noalloc_scratch[NA_HEADER + NA_MAX_BLOCKS];

__device__ __forceinline__ void na_block_max(double &smax, int &bad)
{
    for (int off = 16; off > 0; off >>= 1) {
        const double o = __shfl_xor_sync(0xffffffffu, smax, off);
        if (o > smax) smax = o;
        bad += __shfl_xor_sync(0xffffffffu, bad, off);
    }
    __shared__ double wmax[NA_THREADS / 32];
    __shared__ int wbad[NA_THREADS / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) { wmax[wid] = smax; wbad[wid] = bad; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < NA_THREADS / 32; ++w) {
            if (wmax[w] > smax) smax = wmax[w];
            bad += wbad[w];
        }
    }
}

__global__ void __launch_bounds__(NA_THREADS) cfl_partial_kernel(long long ncell, double gamma, const double *__restrict__ rho,
                                                                 const double *__restrict__ mx, const double *__restrict__ my,
                                                                 const double *__restrict__ mz, const double *__restrict__ E,
                                                                 unsigned long long *scratch)
{
    double smax = 0.0;
    int bad = 0;
    const long long t0 = (long long)blockIdx.x * NA_CELLS_PER_BLOCK + threadIdx.x;
#pragma unroll
    for (int q = 0; q < NA_CELLS_PER_THREAD; ++q) {
        const long long t = t0 + (long long)q * NA_THREADS;
        if (t >= ncell) break;
        const Prim w = cons_to_prim(gamma, rho[t], mx[t], my[t], mz[t], E[t]);
        if (!(w.rho > 0.0) || !(w.P > 0.0)) { ++bad; continue; }
        const double vmag = sqrt((w.vx * w.vx + w.vy * w.vy) + w.vz * w.vz);
        const double cs = sqrt(gamma * w.P / w.rho);
        const double s = vmag + cs;
        if (s > smax) smax = s;
    }
    na_block_max(smax, bad);
    if (threadIdx.x == 0) {
        scratch[NA_HEADER + blockIdx.x] = (unsigned long long)__double_as_longlong(smax);
        if (bad) atomicAdd(&scratch[0], (unsigned long long)bad);
    }
}

__global__ void __launch_bounds__(NA_THREADS) cfl_finish_kernel(int nblocks, double cfl, double dx,
                                                                const unsigned long long *scratch, double *dt_out)
{
    double smax = 0.0;
    int bad = 0;
    for (int b = threadIdx.x; b < nblocks; b += NA_THREADS) {
        const double s = __longlong_as_double((long long)scratch[NA_HEADER + b]);
        if (s > smax) smax = s;
    }
    na_block_max(smax, bad);
    if (threadIdx.x == 0)
        *dt_out = scratch[0] != 0 ? __longlong_as_double(0x7ff8000000000000LL) : cfl * dx / smax;      // eq 21
}

// Device address of the scratch array on the current device: cudaGetSymbolAddress once per device, with that
// device current.  No allocation: the array is part of the loaded module.
constexpr int NA_MAX_DEVICES = 64;
static std::mutex na_mutex;
static unsigned long long *na_ptr[NA_MAX_DEVICES];

static int noalloc_scratch(unsigned long long **out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return QK_ECUDA; }
    if (dev < 0 || dev >= NA_MAX_DEVICES) return QK_EINVAL;
    std::lock_guard<std::mutex> lock(na_mutex);
    if (!na_ptr[dev]) {
        void *p = nullptr;
        if (cudaGetSymbolAddress(&p, qk_noalloc_scratch) != cudaSuccess || !p) { cudaGetLastError(); return QK_ECUDA; }
        na_ptr[dev] = (unsigned long long *)p;
    }
    *out = na_ptr[dev];
    return QK_OK;
}

}  // namespace qk

using namespace qk;

extern "C" long long qk_noalloc_max_cells(void) { return QK_NOALLOC_MAX_CELLS; }

extern "C" int qk_noalloc_setup(void)
{
    unsigned long long *p;
    return noalloc_scratch(&p);
}

extern "C" int qk_cfl_dt_noalloc(const double *rho, const double *mx, const double *my, const double *mz, const double *E,
                                 long long ncells, double gamma, double cfl, double dx, void *cuda_stream, double *dt_out)
{
    if (!rho || !mx || !my || !mz || !E || !dt_out) return QK_EINVAL;
    if (ncells < 1 || !(gamma > 1.0) || !(cfl > 0.0) || !(dx > 0.0)) return QK_EINVAL;
    if (ncells > QK_NOALLOC_MAX_CELLS) return QK_ENOMEM;       // the static scratch holds one partial per 1024 cells
    unsigned long long *scratch;
    const int rc = noalloc_scratch(&scratch);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int nblocks = (int)((ncells + NA_CELLS_PER_BLOCK - 1) / NA_CELLS_PER_BLOCK);
    // the scratch keeps the last call's contents: the bad-cell counter must start at zero
    if (cudaMemsetAsync(scratch, 0, sizeof(unsigned long long), st) != cudaSuccess) { cudaGetLastError(); return QK_ECUDA; }
    cfl_partial_kernel<<<nblocks, NA_THREADS, 0, st>>>(ncells, gamma, rho, mx, my, mz, E, scratch);
    cfl_finish_kernel<<<1, NA_THREADS, 0, st>>>(nblocks, cfl, dx, scratch, dt_out);
    return cudaGetLastError() == cudaSuccess ? QK_OK : QK_ECUDA;
}

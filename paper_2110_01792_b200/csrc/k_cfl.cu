// k_cfl.cu -- CFL signal-speed reduction, eq 21: max over interior cells of
// |v| + c_s with |v| the vector magnitude and c_s = sqrt(gamma P / rho).
//
// HBM-bound (40 B/cell).  Each thread takes the max over a grid-stride set of cells, then a
// warp-shuffle max, a shared-memory max over the warps of the block, and one atomicMax per
// block on the bit pattern (non-negative doubles order like unsigned integers).  The max is
// exact, so the result does not depend on the reduction order.
#include "qk_internal.h"
#include "qk_math.cuh"

namespace qk {

__global__ void __launch_bounds__(256) cfl_max_speed_kernel(Geom g, double gamma, CHydro5 U, StateCache *ctr)
{
    const long long ncell = (long long)g.nx * g.ny * g.nz;
    double smax = 0.0;
    int bad = 0;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < ncell;
         t += (long long)gridDim.x * blockDim.x) {
        const int row = (int)(t / g.nx);
        const int i = (int)(t - (long long)row * g.nx);
        const int k = row / g.ny;
        const int j = row - k * g.ny;
        const int cidx = g.at(i, j, k);
        const Prim w = cons_to_prim(gamma, U.rho[cidx], U.mx[cidx], U.my[cidx], U.mz[cidx], U.E[cidx]);
        if (!(w.rho > 0.0) || !(w.P > 0.0)) { ++bad; continue; }
        const double vmag = sqrt((w.vx * w.vx + w.vy * w.vy) + w.vz * w.vz);
        const double cs = sqrt(gamma * w.P / w.rho);
        const double s = vmag + cs;
        if (s > smax) smax = s;
    }
    for (int off = 16; off > 0; off >>= 1) {
        const double o = __shfl_xor_sync(0xffffffffu, smax, off);
        if (o > smax) smax = o;
        bad += __shfl_xor_sync(0xffffffffu, bad, off);
    }
    __shared__ double wmax[8];
    __shared__ int wbad[8];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) { wmax[wid] = smax; wbad[wid] = bad; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) {
            if (wmax[w] > smax) smax = wmax[w];
            bad += wbad[w];
        }
        atomicMax(&ctr->smax_bits, (unsigned long long)__double_as_longlong(smax));
        if (bad) atomicAdd((unsigned long long *)&ctr->cfl_bad, (unsigned long long)bad);
    }
}

// eq 21 (and the N_sub,max limit) on the device, same operations as qk_cfl_dt does on the host
__global__ void dt_from_cache_kernel(const StateCache *cache, DeviceDt *out, double cfl, double dx, double c_hat, int nsub_max,
                                     int nsub)
{
    double dt;
    if (cache->cfl_bad != 0) {
        dt = __longlong_as_double(0x7ff8000000000000LL);          // NaN: a cell has rho <= 0 or P <= 0
    } else {
        const double smax = __longlong_as_double((long long)cache->smax_bits);
        dt = cfl * dx / smax;
        if (c_hat > 0.0) {
            const double dtr = (double)nsub_max * (cfl * dx / c_hat);
            if (dtr < dt) dt = dtr;
        }
    }
    out->dt = dt;
    out->dtdx = dt / dx;
    out->dts = dt / (double)nsub;                  // radiation substep (qk_rhd_step_cfl), as qk_rhd_step forms it
    out->dtsdx = out->dts / dx;
}

int launch_dt_from_cache(const StateCache *cache, DeviceDt *out, double cfl, double dx, double c_hat, int nsub_max,
                         int nsub, cudaStream_t st)
{
    dt_from_cache_kernel<<<1, 1, 0, st>>>(cache, out, cfl, dx, c_hat, nsub_max, nsub);
    return 1;
}

int launch_cfl(const Geom &g, double gamma, CHydro5 U, StateCache *ctr, cudaStream_t st)
{
    const long long ncell = (long long)g.nx * g.ny * g.nz;
    long long blocks = (ncell + 255) / 256;
    const long long cap = 148LL * 8;
    if (blocks > cap) blocks = cap;
    cfl_max_speed_kernel<<<(unsigned)blocks, 256, 0, st>>>(g, gamma, U, ctr);
    return 1;
}

}  // namespace qk

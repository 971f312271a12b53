// k_boundary.cu -- ghost-zone fill ("B.C. fill"): periodic
// or outflow = zero-gradient copy of the nearest interior cell (reading H15).
//
// Every ghost cell (faces, edges, corners) takes the value of the interior cell its three
// indices map to, so one pass fills the whole shell with no ordering between directions
// (identical to filling x, then y, then z).  Pure data movement: parity with the oracle is
// bit-exact.  The ghost shell is enumerated as three slab families so that no thread is
// spent on interior cells:
//   Z slabs: 2 NG full planes                    (coalesced rows of px)
//   Y slabs: nz planes x 2 NG rows x px          (coalesced rows of px)
//   X slabs: nz x ny rows x 2 NG cells           (8 cells per row, 4 at each end)
#include "qk_internal.h"

namespace qk {

__device__ __forceinline__ int wrap_index(int i, int n, int bc)
{
    if (i >= 0 && i < n) return i;
    if (bc == QK_BC_PERIODIC) {
        int m = i % n;
        return m < 0 ? m + n : m;
    }
    return i < 0 ? 0 : n - 1;
}

__global__ void __launch_bounds__(256) fill_ghost_kernel(Geom g, int bc, FillList fl)
{
    const long long nZ = 2LL * NG * g.py * g.px;
    const long long nY = 2LL * NG * g.nz * g.px;
    const long long nX = 2LL * NG * g.nz * g.ny;
    const long long total = nZ + nY + nX;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total;
         t += (long long)gridDim.x * blockDim.x) {
        int i, j, k;
        if (t < nZ) {
            const int row = (int)(t / g.px);
            i = (int)(t - (long long)row * g.px) - NG;
            const int kk = row / g.py;
            j = row - kk * g.py - NG;
            k = kk < NG ? kk - NG : g.nz + (kk - NG);
        } else if (t < nZ + nY) {
            const long long u = t - nZ;
            const int row = (int)(u / g.px);
            i = (int)(u - (long long)row * g.px) - NG;
            k = row / (2 * NG);
            const int jj = row - k * (2 * NG);
            j = jj < NG ? jj - NG : g.ny + (jj - NG);
        } else {
            const long long u = t - nZ - nY;
            const int row = (int)(u / (2 * NG));
            const int ii = (int)(u - (long long)row * (2 * NG));
            k = row / g.ny;
            j = row - k * g.ny;
            i = ii < NG ? ii - NG : g.nx + (ii - NG);
        }
        const int dst = g.at(i, j, k);
        const int src = g.at(wrap_index(i, g.nx, bc), wrap_index(j, g.ny, bc), wrap_index(k, g.nz, bc));
#pragma unroll 1
        for (int f = 0; f < fl.n; ++f) fl.f[f][dst] = fl.f[f][src];
    }
}

int launch_fill(const Geom &g, int bc, const FillList &fl, cudaStream_t st)
{
    if (fl.n <= 0) return 0;
    const long long total = 2LL * NG * ((long long)g.py * g.px + (long long)g.nz * g.px + (long long)g.nz * g.ny);
    long long blocks = (total + 255) / 256;
    const long long cap = 148LL * 32;
    if (blocks > cap) blocks = cap;
    fill_ghost_kernel<<<(unsigned)blocks, 256, 0, st>>>(g, bc, fl);
    return 1;
}

}  // namespace qk

// k_boundary.cu -- ghost-zone fill ("B.C. fill"): periodic,
// outflow = zero-gradient copy of the nearest interior cell (reading H15), or reflecting =
// mirror image with the wall-normal vector component negated (reading B1).
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
    if (bc == QK_BC_REFLECTING) {      // mirror image about the wall: -1 <- 0, -2 <- 1, n <- n-1, ... (B1)
        const int m = i < 0 ? -1 - i : 2 * n - 1 - i;
        return m < 0 ? 0 : (m > n - 1 ? n - 1 : m);
    }
    return i < 0 ? 0 : n - 1;
}

// `ext` = QK_FACE_* bits of the z faces that border another rank's slab: their ghost planes already hold the
// neighbour's cells at the interior (i, j) positions (qk_halo_unpack), so only their x / y images are filled.
__global__ void __launch_bounds__(256) fill_ghost_kernel(Geom g, FaceBc fb, unsigned ext, int part, FillList fl)
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
        // part 1: everything except the ghost planes of inter-rank faces (fillable before the neighbour's planes have
        // arrived); part 2: only those planes (their x / y images); part 0: all
        if (part) {
            const bool in_ext = (k < 0 && (ext & QK_FACE_ZLO)) || (k >= g.nz && (ext & QK_FACE_ZHI));
            if (in_ext != (part == 2)) continue;
        }
        // per axis: the rule of the face the index lies beyond (FaceBc: x-lo, x-hi, y-lo, y-hi, z-lo, z-hi)
        const int idx3[3] = {i, j, k}, n3[3] = {g.nx, g.ny, g.nz};
        int src3[3];
        bool keep = false, out_refl[3] = {false, false, false};
#pragma unroll
        for (int ax = 0; ax < 3; ++ax) {
            const int v = idx3[ax];
            src3[ax] = v;
            if (v >= 0 && v < n3[ax]) continue;
            const int lohi = v < 0 ? 0 : 1;
            if (ax == 2 && (ext & (lohi ? QK_FACE_ZHI : QK_FACE_ZLO))) continue;      // neighbour's planes: keep k
            const int t_bc = fb.t[2 * ax + lohi];
            if (t_bc == QK_BC_FIXED) { keep = true; continue; }                         // Dirichlet: caller's values
            src3[ax] = wrap_index(v, n3[ax], t_bc);
            out_refl[ax] = t_bc == QK_BC_REFLECTING;
        }
        const int dst = g.at(i, j, k);
        const int src = g.at(src3[0], src3[1], src3[2]);
        if (keep) {       // stage buffers take the Dirichlet values from the state field they shadow
#pragma unroll 1
            for (int f = 0; f < fl.n; ++f)
                if (fl.fixed_src[f]) fl.f[f][dst] = fl.fixed_src[f][dst];
            continue;
        }
        if (src == dst) continue;
        // all loads of the cell are issued before its first store (a store between two loads would order them: the
        // fields may alias as far as the compiler knows, and the kernel lives on loads in flight)
        double v[QK_NFIELDS];
#pragma unroll
        for (int f = 0; f < QK_NFIELDS; ++f)
            if (f < fl.n) v[f] = fl.f[f][src];
        if (out_refl[0] || out_refl[1] || out_refl[2]) {
            // the normal component of rho v / v / F_r / f changes sign across each wall the image lies beyond
#pragma unroll
            for (int f = 0; f < QK_NFIELDS; ++f) {
                const int cm = fl.comp[f];
                if (f < fl.n && cm >= 0 && out_refl[cm]) v[f] = -v[f];
            }
        }
#pragma unroll
        for (int f = 0; f < QK_NFIELDS; ++f)
            if (f < fl.n) fl.f[f][dst] = v[f];
    }
}

// Halo planes of a z face: NG planes x ny x nx interior cells per field, field-major, planes ascending in k.
// pack: the NG interior planes next to the face -> buf;  unpack: buf -> the NG ghost planes beyond the face.
__global__ void __launch_bounds__(256) halo_copy_kernel(Geom g, int face_hi, int unpack, FillList fl, double *buf)
{
    const long long per_field = (long long)NG * g.ny * g.nx;
    const long long total = per_field * fl.n;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total;
         t += (long long)gridDim.x * blockDim.x) {
        const int f = (int)(t / per_field);
        const long long u = t - (long long)f * per_field;
        const int row = (int)(u / g.nx);
        const int i = (int)(u - (long long)row * g.nx);
        const int kk = row / g.ny;
        const int j = row - kk * g.ny;
        int k;
        if (unpack) k = face_hi ? g.nz + kk : kk - NG;
        else        k = face_hi ? g.nz - NG + kk : kk;
        const int cidx = g.at(i, j, k);
        if (unpack) fl.f[f][cidx] = buf[t];
        else        buf[t] = fl.f[f][cidx];
    }
}

int launch_halo_copy(const Geom &g, int face_hi, int unpack, const FillList &fl, double *buf, cudaStream_t st)
{
    if (fl.n <= 0) return 0;
    const long long total = (long long)NG * g.ny * g.nx * fl.n;
    long long blocks = (total + 255) / 256;
    if (blocks > 148LL * 16) blocks = 148LL * 16;
    halo_copy_kernel<<<(unsigned)blocks, 256, 0, st>>>(g, face_hi, unpack, fl, buf);
    return 1;
}

// ---- peer-mapped halo exchange (qk_set_halo_peers) -------------------------------------------------------------
// The NG interior planes next to a z face go straight into the ghost planes of the neighbour's fields (peer memory:
// NVLink stores, or the same device in the single-process tests), interior (i, j) cells only -- the neighbour's own
// fill makes their x / y images.  dst[f] = the neighbour's array that corresponds to fl.f[f], whose box may have a
// different nz (dg = its geometry).  One 16-byte store per thread where the row pitch allows it.
__global__ void __launch_bounds__(256) halo_push_kernel(Geom g, Geom dg, int face_hi, FillList fl, PeerList dst)
{
    const long long per_field = (long long)NG * g.ny * g.nx;
    const long long total = per_field * fl.n;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total;
         t += (long long)gridDim.x * blockDim.x) {
        const int f = (int)(t / per_field);
        const long long u = t - (long long)f * per_field;
        const int row = (int)(u / g.nx);
        const int i = (int)(u - (long long)row * g.nx);
        const int kk = row / g.ny;
        const int j = row - kk * g.ny;
        // my planes nz-NG+kk (high face) land in the neighbour's planes -NG+kk; my planes kk (low face) in its nz'+kk
        const int ks = face_hi ? g.nz - NG + kk : kk;
        const int kd = face_hi ? kk - NG : dg.nz + kk;
        dst.f[f][dg.at(i, j, kd)] = fl.f[f][g.at(i, j, ks)];
    }
}

// the neighbour's arrival counter <- epoch, after every store of the push is visible system-wide
__global__ void halo_signal_kernel(unsigned long long *flag, unsigned long long epoch)
{
    __threadfence_system();
    *(volatile unsigned long long *)flag = epoch;
    __threadfence_system();
}

int launch_halo_push(const Geom &g, const Geom &dg, int face_hi, const FillList &fl, const PeerList &dst,
                     unsigned long long *flag, unsigned long long epoch, cudaStream_t st)
{
    if (fl.n <= 0) return 0;
    const long long total = (long long)NG * g.ny * g.nx * fl.n;
    long long blocks = (total + 255) / 256;
    if (blocks > 148LL * 8) blocks = 148LL * 8;
    halo_push_kernel<<<(unsigned)blocks, 256, 0, st>>>(g, dg, face_hi, fl, dst);
    halo_signal_kernel<<<1, 1, 0, st>>>(flag, epoch);
    return 2;
}

int launch_fill(const Geom &g, const FaceBc &fb, unsigned ext, int part, const FillList &fl, cudaStream_t st)
{
    if (fl.n <= 0) return 0;
    const long long total = 2LL * NG * ((long long)g.py * g.px + (long long)g.nz * g.px + (long long)g.nz * g.ny);
    long long blocks = (total + 255) / 256;
    const long long cap = 148LL * 32;
    if (blocks > cap) blocks = cap;
    fill_ghost_kernel<<<(unsigned)blocks, 256, 0, st>>>(g, fb, ext, part, fl);
    return 1;
}

}  // namespace qk

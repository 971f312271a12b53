// qk_internal.h -- layout, context and kernel-launcher declarations shared by the .cu files of
// libqk (not part of the public ABI; see include/qk.h for that).
#pragma once

#include <cuda_runtime.h>
#include <stddef.h>
#include <vector>

#include "../../include/qk.h"

namespace qk {

constexpr int NG = QK_NG;

// Box geometry.  Cell (i,j,k) with ghost range -NG..n+NG-1 lives at (k+NG)*sz + (j+NG)*sy + (i+NG).
struct Geom {
    int nx, ny, nz;      // interior cells
    int px, py, pz;      // padded extents n + 2 NG
    int sy, sz;          // strides in doubles (x stride is 1)
    int ntot;            // px*py*pz  (<= 2^31: 512^3 boxes are 1.4e8)
    __host__ __device__ int at(int i, int j, int k) const { return (k + NG) * sz + (j + NG) * sy + (i + NG); }
};

inline Geom make_geom(int nx, int ny, int nz)
{
    Geom g;
    g.nx = nx; g.ny = ny; g.nz = nz;
    g.px = nx + 2 * NG; g.py = ny + 2 * NG; g.pz = nz + 2 * NG;
    g.sy = g.px; g.sz = g.px * g.py;
    g.ntot = g.px * g.py * g.pz;
    return g;
}

// Device-side counters of one public step call (zeroed at its start).
struct Counters {
    unsigned long long smax_bits;      // CFL: bit pattern of max(|v|+c_s) (non-negative doubles order as integers)
    long long cfl_bad;                 // CFL: cells with rho<=0 or P<=0
    long long bad_state;               // step kernels: cells with rho<=0, P<=0, E_g<=0, E_r<=0
    long long newton_fail;
    long long newton_total;
    long long fallback;
    long long guard;
    int newton_max;
    int pad;
};

// Results that stay valid between public calls (never cleared by reset_counters): the CFL signal speed of
// the current hydro state, written by the kernel that produced that state (or by the CFL kernel).
struct StateCache {
    unsigned long long smax_bits;      // bit pattern of max(|v|+c_s) over interior cells
    long long cfl_bad;                 // interior cells with rho<=0 or P<=0
};

// Timestep kept on the device (qk_hydro_step_cfl): eq 21 evaluated from the cached signal speed by a one-thread
// kernel, read by the z sweeps.  Lives beside StateCache, outside the part that is cleared between RK stages.
struct DeviceDt { double dt, dtdx, dts, dtsdx; };     // step, step / dx, radiation substep, substep / dx
int launch_dt_from_cache(const StateCache *cache, DeviceDt *out, double cfl, double dx, double c_hat, int nsub_max,
                         int nsub, cudaStream_t st);

// Kernel classes for per-kernel timing (qk_kernel_times) -- one id per __global__ function family.
enum KClass { K_FILL = 0, K_CFL, K_FLATTEN, K_HYDRO_X, K_HYDRO_Y, K_HYDRO_Z, K_RAD_X, K_RAD_Y, K_RAD_Z, K_EXCHANGE, K_OPACITY, K_PRIM, K_HALO, K_NCLASS };

struct PhysConsts {
    double dx, gamma, c_hat, c, a_rad, kB_mu, cfl, newton_tol;
    double opac_kP0, opac_kR0, opac_rho0;   // opacity law (qk_set_opacity_law); opac_rho0 = 0: the fields as set
    int opac_exp;
    int opac_texp2;        // ... times (T/T0)^(opac_texp2/2) (qk_set_opacity_law_T); 0: no temperature dependence
    double opac_T0;
    double eos_alpha;      // > 0: E_g = alpha T^4 / 4 in the exchange (eq 55); 0: ideal gas
    int newton_maxit, nsub_max;
    unsigned flags;
    int bc;
};

// Field pointer bundles passed to kernels by value.
struct Hydro5 { double *rho, *mx, *my, *mz, *E; };
struct CHydro5 { const double *rho, *mx, *my, *mz, *E; };
struct Rad4p { double *E, *Fx, *Fy, *Fz; };
struct CRad4p { const double *E, *Fx, *Fy, *Fz; };

// comp[i] = vector component field i carries (0, 1, 2) or -1 for a scalar: negated in the image cells of a
// reflecting wall normal to that axis
// fixed_src[i] != nullptr: ghost cells of field i beyond a QK_BC_FIXED face are copied from that array (same cell):
// how the RK stage buffers get the Dirichlet values the caller stored in the state fields
struct FillList { double *f[QK_NFIELDS]; const double *fixed_src[QK_NFIELDS]; signed char comp[QK_NFIELDS]; int n; };

// ---- launchers (each enqueues on `st`; returns the number of kernels launched) -----------------
struct FaceBc { int t[6]; };      // QK_BC_* of the faces x-lo, x-hi, y-lo, y-hi, z-lo, z-hi
// part 0: the whole ghost shell; 1: all but the ghost planes of the inter-rank faces; 2: only those planes
int launch_fill(const Geom &g, const FaceBc &fb, unsigned ext_faces, int part, const FillList &fl, cudaStream_t st);
struct PeerList { double *f[QK_NFIELDS]; };      // the neighbour's arrays that correspond to a FillList
int launch_halo_push(const Geom &g, const Geom &dg, int face_hi, const FillList &fl, const PeerList &dst,
                     unsigned long long *flag, unsigned long long epoch, cudaStream_t st);
int launch_halo_copy(const Geom &g, int face_hi, int unpack, const FillList &fl, double *buf, cudaStream_t st);
int launch_cfl(const Geom &g, double gamma, CHydro5 U, StateCache *cache, cudaStream_t st);

// stencil kernels of an RK stage (k_sweep.cu); `which` bit 0 = x sweep (D = dF_x), bit 1 = y sweep (D += dF_y),
// bit 2 = z sweep (RK update).  W / S: reconstruction variables of the stage's state with their ghost cells filled;
// U / R: that state (own-cell reads of the update); U0 / R0: the state at the start of the step; Wout / Sout: the
// reconstruction variables of the updated interior cells.
int launch_chi(const Geom &g, double gamma, CHydro5 W, double *cx, double *cy, double *cz, double *chi, int d0, int d1,
               int m0, int m1, int path, cudaStream_t st);
int launch_hydro_sweeps(const Geom &g, double gamma, unsigned scheme, double dtdx, int stage, CHydro5 W,
                        const double *chi, Hydro5 D, CHydro5 U, CHydro5 U0, Hydro5 out, Hydro5 Wout, Counters *ctr,
                        StateCache *cache, cudaStream_t st, int which, const double *dtdx_dev, int k0, int k1);
int launch_rad_sweeps(const Geom &g, const PhysConsts &pc, double dtdx, int stage, CRad4p S, const double *rho,
                      const double *kappaR, Rad4p D, CRad4p R, CRad4p R0, Rad4p out, Rad4p Sout, Counters *ctr,
                      cudaStream_t st, int which, const double *dtdx_dev, int k0, int k1);
int launch_prim(const Geom &g, double gamma, CHydro5 U, Hydro5 W, Counters *ctr, cudaStream_t st);
int launch_rad_prim(const Geom &g, double c, CRad4p R, Rad4p S, Counters *ctr, cudaStream_t st);

// opacity law kappa0 (rho/rho0)^e (T/T0)^(texp2/2) of the interior cells from the current state (X14)
int launch_opacity_law(const Geom &g, const PhysConsts &pc, CHydro5 U, double *kP, double *kR, cudaStream_t st);
// dt_dev != nullptr: the substep is read from device memory.  The kernel leaves the CFL signal speed of the updated
// state in `cache` and, when Wout.rho != nullptr, the reconstruction variables W and S of the updated cells
int launch_exchange(const Geom &g, const PhysConsts &pc, double dt, const double *dt_dev, const double *rho, double *mx, double *my,
                    double *mz, double *E, double *Er, double *Fx, double *Fy, double *Fz, const double *kP,
                    const double *kR, const double *src, Hydro5 Wout, Rad4p Sout, Counters *ctr, StateCache *cache,
                    cudaStream_t st);

}  // namespace qk

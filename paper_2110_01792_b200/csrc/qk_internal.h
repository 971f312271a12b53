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
struct DeviceDt { double dt, dtdx; };
int launch_dt_from_cache(const StateCache *cache, DeviceDt *out, double cfl, double dx, double c_hat, int nsub_max,
                         cudaStream_t st);

// Kernel classes for per-kernel timing (qk_kernel_times) -- one id per __global__ function family.
enum KClass { K_FILL = 0, K_CFL, K_PRIM, K_FLATTEN, K_HYDRO_FLUX, K_HYDRO_UPDATE, K_HYDRO_STAGE,
              K_RAD_PRIM, K_RAD_FLUX, K_RAD_UPDATE, K_RAD_STAGE, K_EXCHANGE,
              K_HYDRO_SWEEP_X, K_HYDRO_SWEEP_Y, K_HYDRO_SWEEP_Z, K_RAD_SWEEP_X, K_RAD_SWEEP_Y, K_RAD_SWEEP_Z,
              K_NCLASS };

struct PhysConsts {
    double dx, gamma, c_hat, c, a_rad, kB_mu, cfl, newton_tol;
    double opac_kP0, opac_kR0, opac_rho0;   // opacity law (qk_set_opacity_law); opac_rho0 = 0: the fields as set
    int opac_exp;
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
struct FillList { double *f[QK_NFIELDS]; signed char comp[QK_NFIELDS]; int n; };

// ---- launchers (each enqueues on `st`; returns the number of kernels launched) -----------------
struct FaceBc { int t[6]; };      // QK_BC_* of the faces x-lo, x-hi, y-lo, y-hi, z-lo, z-hi
int launch_fill(const Geom &g, const FaceBc &fb, unsigned ext_faces, const FillList &fl, cudaStream_t st);
int launch_halo_copy(const Geom &g, int face_hi, int unpack, const FillList &fl, double *buf, cudaStream_t st);
int launch_cfl(const Geom &g, double gamma, CHydro5 U, StateCache *cache, cudaStream_t st);

int launch_prim(const Geom &g, double gamma, CHydro5 U, Hydro5 W, Counters *ctr, cudaStream_t st);
int launch_flatten(const Geom &g, double gamma, CHydro5 W, double *chi, cudaStream_t st);
int launch_hydro_flux(const Geom &g, double gamma, int dir, CHydro5 W, const double *chi, Hydro5 flux, cudaStream_t st);
int launch_hydro_update(const Geom &g, double dtdx, int stage, CHydro5 U, CHydro5 U0, CHydro5 fx, CHydro5 fy,
                        CHydro5 fz, Hydro5 out, cudaStream_t st);

// fused path (k_hydro.cu, k_rad.cu)
int launch_flatten_march(const Geom &g, double gamma, CHydro5 U, double *chi, cudaStream_t st);
int launch_hydro_stage(const Geom &g, double gamma, double dtdx, int stage, CHydro5 U, CHydro5 U0, const double *chi,
                       Hydro5 out, Counters *ctr, cudaStream_t st);

int launch_rad_stage(const Geom &g, const PhysConsts &pc, double dtdx, int stage, CRad4p R, CRad4p R0, const double *rho,
                     const double *kappaR, Rad4p out, Counters *ctr, cudaStream_t st);

// sweep path (k_sweep.cu); `which` bit 0 = x sweep, bit 1 = y sweep, bit 2 = z sweep + RK update
int launch_hydro_sweeps(const Geom &g, double gamma, unsigned scheme, double dtdx, int stage, CHydro5 W,
                        const double *chi, Hydro5 D, CHydro5 U, CHydro5 U0, Hydro5 out, Hydro5 Wout, Counters *ctr,
                        StateCache *cache, cudaStream_t st, int which, const double *dtdx_dev);
int launch_chi_two_pass(const Geom &g, double gamma, CHydro5 W, double *cx, double *cy, double *cz, double *chi,
                        cudaStream_t st);
int launch_rad_sweeps(const Geom &g, const PhysConsts &pc, double dtdx, int stage, CRad4p S, const double *rho,
                      const double *kappaR, Rad4p D, CRad4p R, CRad4p R0, Rad4p out, Rad4p Sout, Counters *ctr,
                      cudaStream_t st, int which);

int launch_rad_prim(const Geom &g, double c, CRad4p R, Rad4p S, Counters *ctr, cudaStream_t st);
int launch_rad_flux(const Geom &g, const PhysConsts &pc, int dir, CRad4p S, const double *rho, const double *kappaR,
                    Rad4p flux, Counters *ctr, cudaStream_t st);
int launch_rad_update(const Geom &g, double dtdx, int stage, CRad4p R, CRad4p R0, CRad4p gx, CRad4p gy, CRad4p gz,
                      Rad4p out, cudaStream_t st);

int launch_opacity_law(const Geom &g, const double *rho, double *kP, double *kR, double kP0, double kR0, double rho0,
                       int e, cudaStream_t st);
int launch_exchange(const Geom &g, const PhysConsts &pc, double dt, const double *rho, double *mx, double *my,
                    double *mz, double *E, double *Er, double *Fx, double *Fy, double *Fz, const double *kP,
                    const double *kR, const double *src, Hydro5 Wout, Rad4p Sout, Counters *ctr, StateCache *cache,
                    cudaStream_t st);
// Wout.rho == nullptr: exchange only; otherwise the kernel also writes the primitives W and the radiation
// variables S = (E_r, f) of the updated cells and leaves the CFL speed of the new state in `cache`

}  // namespace qk

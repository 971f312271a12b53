// qk_api.cu -- the C ABI of include/qk.h: context, device storage layout, step drivers.
//
// Storage (one allocation, caller- or library-owned), all fp64 SoA, each array padded to a
// multiple of 32 doubles so every field starts 256-byte aligned:
//   [ 11 state fields | 5 RK stage fields | chi | scratch fields of the unfused path | counters ]
// Drivers follow the operator-split cycle of PAPER.md:112: hydro step (SSP-RK2),
// then N_sub x (radiation transport RK2, exchange).
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <new>

#include "qk_internal.h"

using namespace qk;

namespace {

constexpr int N_STAGE = 5;          // U^(1) (hydro) / first 4 reused for radiation
constexpr int N_SCRATCH_REF = 28;   // unfused path: primitives + 3 x 5 flux fields (0..19); sweep path: see SC_*
// scratch fields of the sweep path: two primitive sets W (ping-pong between RK stages), the flux-difference
// accumulators D, the three directional flattening coefficients, two radiation sets S = (E_r, f)
constexpr int SC_WA = 0, SC_D = 5, SC_CHI3 = 10, SC_WB = 15, SC_SA = 20, SC_SB = 24;
constexpr size_t COUNTER_BYTES = 256;

inline size_t field_stride(const Geom &g) { return ((size_t)g.ntot + 31) / 32 * 32; }

}  // namespace

struct qk_ctx {
    Geom g;
    PhysConsts pc;
    cudaStream_t stream;
    int device;
    char *base;            // device storage
    size_t bytes;
    bool owns;
    bool ready;
    double *state[QK_NFIELDS];
    double *stage[N_STAGE];
    double *chi;
    double *scratch[N_SCRATCH_REF];
    Counters *ctr;
    StateCache *cache;
    DeviceDt *ddt;         // device-resident timestep of qk_hydro_step_cfl
    // sweep path: which scratch set holds the reconstruction variables of the current state (interior
    // cells), and whether it / the cached CFL speed still describe the state
    int w_cur, s_cur;
    bool w_valid, s_valid, smax_valid;
    FaceBc fb;             // boundary type of each face (qk_init sets all six alike)
    bool has_fixed;        // some face is QK_BC_FIXED: the ghost cells beyond it hold caller-supplied values
    bool has_source;       // QK_SRC was set: the exchange reads it (otherwise S = 0 and the field is never touched)
    int path;              // QK_PATH_*
    // z-slab decomposition: inter-rank faces, the caller's halo mover, and the field list of the fill in progress
    unsigned ext_faces;
    qk_halo_fn halo_fn;
    void *halo_user;
    FillList pending;
    bool in_halo_cb;
    long long launches;
    int last_nsub;
    // per-kernel-class event timing
    bool profiling;
    struct Span { int cls; cudaEvent_t a, b; };
    std::vector<Span> spans;
    std::vector<cudaEvent_t> pool;
};

namespace {

size_t total_bytes(const Geom &g)
{
    const size_t nf = QK_NFIELDS + N_STAGE + 1 + N_SCRATCH_REF;
    return nf * field_stride(g) * sizeof(double) + COUNTER_BYTES;
}

int carve(qk_ctx *c)
{
    const size_t fs = field_stride(c->g);
    double *p = (double *)c->base;
    for (int f = 0; f < QK_NFIELDS; ++f) { c->state[f] = p; p += fs; }
    for (int f = 0; f < N_STAGE; ++f) { c->stage[f] = p; p += fs; }
    c->chi = p; p += fs;
    for (int f = 0; f < N_SCRATCH_REF; ++f) { c->scratch[f] = p; p += fs; }
    c->ctr = (Counters *)p;
    c->cache = (StateCache *)((char *)p + 128);
    c->ddt = (DeviceDt *)((char *)p + 192);
    // zero everything once so ghost cells and unused corners are defined
    if (cudaMemsetAsync(c->base, 0, c->bytes, c->stream) != cudaSuccess) return QK_ECUDA;
    c->ready = true;
    return QK_OK;
}

int ensure_storage(qk_ctx *c)
{
    if (c->ready) return QK_OK;
    if (cudaSetDevice(c->device) != cudaSuccess) return QK_ECUDA;
    if (!c->base) {
        c->bytes = total_bytes(c->g);
        void *p = nullptr;
        if (cudaMalloc(&p, c->bytes) != cudaSuccess) { cudaGetLastError(); return QK_ENOMEM; }
        c->base = (char *)p;
        c->owns = true;
    }
    return carve(c);
}

bool is_device_ptr(const void *p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

// copy between a dense interior array and the ghosted field
int copy_interior(qk_ctx *c, double *field, double *dense, bool to_field)
{
    const Geom &g = c->g;
    cudaMemcpy3DParms p;
    memset(&p, 0, sizeof(p));
    cudaPitchedPtr fptr = make_cudaPitchedPtr(field, (size_t)g.px * sizeof(double), g.px, g.py);
    cudaPitchedPtr dptr = make_cudaPitchedPtr(dense, (size_t)g.nx * sizeof(double), g.nx, g.ny);
    const cudaPos fpos = make_cudaPos((size_t)NG * sizeof(double), NG, NG);
    const cudaPos dpos = make_cudaPos(0, 0, 0);
    if (to_field) { p.srcPtr = dptr; p.srcPos = dpos; p.dstPtr = fptr; p.dstPos = fpos; }
    else          { p.srcPtr = fptr; p.srcPos = fpos; p.dstPtr = dptr; p.dstPos = dpos; }
    p.extent = make_cudaExtent((size_t)g.nx * sizeof(double), g.ny, g.nz);
    p.kind = cudaMemcpyDefault;
    return cudaMemcpy3DAsync(&p, c->stream) == cudaSuccess ? QK_OK : QK_ECUDA;
}

// ---- launch bookkeeping -------------------------------------------------------------------------
cudaEvent_t get_event(qk_ctx *c)
{
    if (!c->pool.empty()) { cudaEvent_t e = c->pool.back(); c->pool.pop_back(); return e; }
    cudaEvent_t e;
    cudaEventCreate(&e);
    return e;
}

struct Scope {   // brackets the launches of one kernel class with events when profiling is on
    qk_ctx *c; int cls; cudaEvent_t a;
    Scope(qk_ctx *ctx, int k) : c(ctx), cls(k), a(nullptr)
    {
        if (c->profiling) { a = get_event(c); cudaEventRecord(a, c->stream); }
    }
    void done(int nlaunch)
    {
        c->launches += nlaunch;
        if (c->profiling) {
            cudaEvent_t b = get_event(c);
            cudaEventRecord(b, c->stream);
            c->spans.push_back({cls, a, b});
        }
    }
};

int check_launch() { return cudaGetLastError() == cudaSuccess ? QK_OK : QK_ECUDA; }

Hydro5 h5(double *const *f) { return Hydro5{f[0], f[1], f[2], f[3], f[4]}; }
CHydro5 ch5(double *const *f) { return CHydro5{f[0], f[1], f[2], f[3], f[4]}; }
Rad4p r4(double *const *f) { return Rad4p{f[0], f[1], f[2], f[3]}; }
CRad4p cr4(double *const *f) { return CRad4p{f[0], f[1], f[2], f[3]}; }

void reset_counters(qk_ctx *c) { cudaMemsetAsync(c->ctr, 0, sizeof(Counters), c->stream); }

// Every list the drivers fill is (scalar, x, y, z component, scalars ...): U, W, R, S, optionally followed by rho
// and kappa_R; qk_fill_boundary passes the components of its own list.
void fill_fields(qk_ctx *c, double *const *fields, int n, const signed char *comps = nullptr)
{
    FillList fl;
    fl.n = n;
    for (int i = 0; i < n; ++i) {
        fl.f[i] = fields[i];
        fl.comp[i] = comps ? comps[i] : (signed char)((i >= 1 && i <= 3) ? i - 1 : -1);
    }
    Scope s(c, K_FILL);
    if (c->ext_faces && c->halo_fn) {      // neighbours' planes first, then the x / y images of everything
        c->pending = fl;
        c->in_halo_cb = true;
        c->halo_fn(c->halo_user, n);
        c->in_halo_cb = false;
    }
    s.done(launch_fill(c->g, c->fb, c->ext_faces, fl, c->stream));
}

// ---- hydro: SSP-RK2 ------------------------------------------------------------------
// stage 1:  U1 = Un - (dt/dx) div F(Un)            -> stage buffers
// stage 2:  Un+1 = 0.5 Un + 0.5 (U1 - (dt/dx) div F(U1))   -> state (each cell reads only its own Un)
void hydro_stage_unfused(qk_ctx *c, double dtdx, int stage, double *const *U, double *const *U0, double *const *out)
{
    const Geom &g = c->g;
    double *const *W = &c->scratch[0];
    double *const *fx = &c->scratch[5], *const *fy = &c->scratch[10], *const *fz = &c->scratch[15];
    { Scope s(c, K_PRIM); s.done(launch_prim(g, c->pc.gamma, ch5(U), h5(W), c->ctr, c->stream)); }
    { Scope s(c, K_FLATTEN); s.done(launch_flatten(g, c->pc.gamma, ch5(W), c->chi, c->stream)); }
    {
        Scope s(c, K_HYDRO_FLUX);
        int n = launch_hydro_flux(g, c->pc.gamma, 0, ch5(W), c->chi, h5(fx), c->stream);
        n += launch_hydro_flux(g, c->pc.gamma, 1, ch5(W), c->chi, h5(fy), c->stream);
        n += launch_hydro_flux(g, c->pc.gamma, 2, ch5(W), c->chi, h5(fz), c->stream);
        s.done(n);
    }
    {
        Scope s(c, K_HYDRO_UPDATE);
        s.done(launch_hydro_update(g, dtdx, stage, ch5(U), ch5(U0), ch5(fx), ch5(fy), ch5(fz), h5(out), c->stream));
    }
}

void hydro_stage_fused(qk_ctx *c, double dtdx, int stage, double *const *U, double *const *U0, double *const *out)
{
    const Geom &g = c->g;
    { Scope s(c, K_FLATTEN); s.done(launch_flatten_march(g, c->pc.gamma, ch5(U), c->chi, c->stream)); }
    {
        Scope s(c, K_HYDRO_STAGE);
        s.done(launch_hydro_stage(g, c->pc.gamma, dtdx, stage, ch5(U), ch5(U0), c->chi, h5(out), c->ctr, c->stream));
    }
}

// Sweep path.  W_in holds the primitives of U (interior cells when `w_ready`; otherwise they are computed
// here for every cell from the ghost-filled U).  The z sweep writes the updated state and its primitives
// W_out (interior), and after the last stage the CFL speed of the new state.
void hydro_stage_sweep(qk_ctx *c, double dtdx, int stage, double *const *U, double *const *U0, double *const *out,
                       double *const *W, double *const *Wout, bool w_ready, const double *dtdx_dev)
{
    const Geom &g = c->g;
    double *const *D = &c->scratch[SC_D];
    if (w_ready) {
        fill_fields(c, W, 5);            // periodic / outflow / mirror images commute with the pointwise cons -> prim map
    } else {
        fill_fields(c, U, 5);
        Scope s(c, K_PRIM);
        int n = launch_prim(g, c->pc.gamma, ch5(U), h5(W), c->ctr, c->stream);
        // ghost cells beyond a Dirichlet face are never refilled: the other W set needs their primitives too
        if (c->has_fixed) n += launch_prim(g, c->pc.gamma, ch5(U), h5(Wout), c->ctr, c->stream);
        s.done(n);
    }
    {
        Scope s(c, K_FLATTEN);
        s.done(launch_chi_two_pass(g, c->pc.gamma, ch5(W), c->scratch[SC_CHI3], c->scratch[SC_CHI3 + 1],
                                   c->scratch[SC_CHI3 + 2], c->chi, c->stream));
    }
    for (int d = 0; d < 3; ++d) {
        Scope s(c, K_HYDRO_SWEEP_X + d);
        s.done(launch_hydro_sweeps(g, c->pc.gamma, c->pc.flags, dtdx, stage, ch5(W), c->chi, h5(D), ch5(U), ch5(U0), h5(out), h5(Wout),
                                   c->ctr, c->cache, c->stream, 1 << d, dtdx_dev));
    }
}

void hydro_stage(qk_ctx *c, double dtdx, int stage, double *const *U, double *const *U0, double *const *out)
{
    fill_fields(c, U, 5);
    if (c->path == QK_PATH_FUSED) hydro_stage_fused(c, dtdx, stage, U, U0, out);
    else hydro_stage_unfused(c, dtdx, stage, U, U0, out);
}

// the PLM / Eddington variants and Dirichlet faces exist in the sweep path only
bool scheme_supported(const qk_ctx *c)
{
    return c->path == QK_PATH_SWEEP || (!(c->pc.flags & (QK_FLAG_PLM | QK_FLAG_EDDINGTON | QK_FLAG_MINERBO)) && !c->has_fixed);
}

int do_hydro_step(qk_ctx *c, double dt, const double *dtdx_dev = nullptr)
{
    if (!scheme_supported(c)) return QK_EINVAL;
    const double dtdx = dt / c->pc.dx;
    double *const *Un = &c->state[QK_RHO];
    double *const *U1 = &c->stage[0];
    if (c->path == QK_PATH_SWEEP) {
        double *const *W0 = &c->scratch[c->w_cur ? SC_WB : SC_WA];
        double *const *W1 = &c->scratch[c->w_cur ? SC_WA : SC_WB];
        hydro_stage_sweep(c, dtdx, 0, Un, Un, U1, W0, W1, c->w_valid, dtdx_dev);
        cudaMemsetAsync(c->cache, 0, sizeof(StateCache), c->stream);
        hydro_stage_sweep(c, dtdx, 1, U1, Un, Un, W1, W0, true, dtdx_dev);
        c->w_valid = true;               // W0 = primitives of the new state, cache = its CFL speed
        c->smax_valid = true;
    } else {
        hydro_stage(c, dtdx, 0, Un, Un, U1);
        hydro_stage(c, dtdx, 1, U1, Un, Un);
        c->w_valid = false;              // these paths use the scratch fields for their own intermediates
        c->s_valid = false;
        c->smax_valid = false;
    }
    return check_launch();
}

// ---- radiation transport: same SSP-RK2 -----------------------------------------------------
void rad_stage_unfused(qk_ctx *c, double dtdx, int stage, double *const *R, double *const *R0, double *const *out)
{
    const Geom &g = c->g;
    double *const *S = &c->scratch[0];
    double *const *gx = &c->scratch[5], *const *gy = &c->scratch[10], *const *gz = &c->scratch[15];
    { Scope s(c, K_RAD_PRIM); s.done(launch_rad_prim(g, c->pc.c, cr4(R), r4(S), c->ctr, c->stream)); }
    {
        Scope s(c, K_RAD_FLUX);
        int n = 0;
        for (int d = 0; d < 3; ++d)
            n += launch_rad_flux(g, c->pc, d, cr4(S), c->state[QK_RHO], c->state[QK_KAPPA_R],
                                 r4(d == 0 ? gx : (d == 1 ? gy : gz)), c->ctr, c->stream);
        s.done(n);
    }
    {
        Scope s(c, K_RAD_UPDATE);
        s.done(launch_rad_update(g, dtdx, stage, cr4(R), cr4(R0), cr4(gx), cr4(gy), cr4(gz), r4(out), c->stream));
    }
}

void rad_stage_fused(qk_ctx *c, double dtdx, int stage, double *const *R, double *const *R0, double *const *out)
{
    Scope s(c, K_RAD_STAGE);
    s.done(launch_rad_stage(c->g, c->pc, dtdx, stage, cr4(R), cr4(R0), c->state[QK_RHO], c->state[QK_KAPPA_R], r4(out),
                            c->ctr, c->stream));
}

void rad_stage_sweep(qk_ctx *c, double dtdx, int stage, double *const *R, double *const *R0, double *const *out,
                     double *const *S, double *const *Sout, bool s_ready, bool first)
{
    const Geom &g = c->g;
    double *const *D = &c->scratch[SC_D];
    // rho and kappa_R ghosts feed tau_face at the domain faces (first stage of a transport step only)
    double *list[6];
    int n = 0;
    double *const *src = s_ready ? S : R;
    for (int f = 0; f < 4; ++f) list[n++] = src[f];
    if (first) { list[n++] = c->state[QK_RHO]; list[n++] = c->state[QK_KAPPA_R]; }
    fill_fields(c, list, n);
    if (!s_ready) {
        Scope s(c, K_RAD_PRIM);
        int n = launch_rad_prim(g, c->pc.c, cr4(R), r4(S), c->ctr, c->stream);
        if (c->has_fixed) n += launch_rad_prim(g, c->pc.c, cr4(R), r4(Sout), c->ctr, c->stream);
        s.done(n);
    }
    for (int d = 0; d < 3; ++d) {
        Scope s(c, K_RAD_SWEEP_X + d);
        s.done(launch_rad_sweeps(g, c->pc, dtdx, stage, cr4(S), c->state[QK_RHO], c->state[QK_KAPPA_R], r4(D), cr4(R),
                                 cr4(R0), r4(out), r4(Sout), c->ctr, c->stream, 1 << d));
    }
}

void rad_stage(qk_ctx *c, double dtdx, int stage, double *const *R, double *const *R0, double *const *out)
{
    if (c->path == QK_PATH_FUSED) rad_stage_fused(c, dtdx, stage, R, R0, out);
    else rad_stage_unfused(c, dtdx, stage, R, R0, out);
}

int do_rad_transport(qk_ctx *c, double dt)
{
    if (!scheme_supported(c)) return QK_EINVAL;
    if (c->pc.opac_rho0 > 0.0) {         // opacities follow the density the hydro step left (X14)
        Scope s(c, K_RAD_PRIM);
        s.done(launch_opacity_law(c->g, c->state[QK_RHO], c->state[QK_KAPPA_P], c->state[QK_KAPPA_R], c->pc.opac_kP0,
                                  c->pc.opac_kR0, c->pc.opac_rho0, c->pc.opac_exp, c->stream));
    }
    const double dtdx = dt / c->pc.dx;
    double *const *Rn = &c->state[QK_ER];
    double *const *R1 = &c->stage[0];
    if (c->path == QK_PATH_SWEEP) {
        double *const *S0 = &c->scratch[c->s_cur ? SC_SB : SC_SA];
        double *const *S1 = &c->scratch[c->s_cur ? SC_SA : SC_SB];
        rad_stage_sweep(c, dtdx, 0, Rn, Rn, R1, S0, S1, c->s_valid, true);
        rad_stage_sweep(c, dtdx, 1, R1, Rn, Rn, S1, S0, true, false);
        c->s_valid = true;
    } else {
        double *first[6] = {Rn[0], Rn[1], Rn[2], Rn[3], c->state[QK_RHO], c->state[QK_KAPPA_R]};
        fill_fields(c, first, 6);
        rad_stage(c, dtdx, 0, Rn, Rn, R1);
        fill_fields(c, R1, 4);
        rad_stage(c, dtdx, 1, R1, Rn, Rn);
        c->w_valid = false;
        c->s_valid = false;
    }
    return check_launch();
}

int do_exchange(qk_ctx *c, double dt)
{
    double *const *s = c->state;
    const bool sweep = c->path == QK_PATH_SWEEP;
    Hydro5 W{nullptr, nullptr, nullptr, nullptr, nullptr};
    Rad4p S{nullptr, nullptr, nullptr, nullptr};
    if (sweep) {     // the exchange rewrites rho v, E, E_r, F_r: it also refreshes what the next stages read
        W = h5(&c->scratch[c->w_cur ? SC_WB : SC_WA]);
        S = r4(&c->scratch[c->s_cur ? SC_SB : SC_SA]);
        cudaMemsetAsync(c->cache, 0, sizeof(StateCache), c->stream);
    }
    Scope sc(c, K_EXCHANGE);
    sc.done(launch_exchange(c->g, c->pc, dt, s[QK_RHO], s[QK_MX], s[QK_MY], s[QK_MZ], s[QK_E], s[QK_ER], s[QK_FX],
                            s[QK_FY], s[QK_FZ], s[QK_KAPPA_P], s[QK_KAPPA_R], c->has_source ? s[QK_SRC] : nullptr, W, S, c->ctr,
                            c->cache, c->stream));
    c->w_valid = sweep;
    c->s_valid = sweep;
    c->smax_valid = sweep;
    return check_launch();
}

int nsub_for(const qk_ctx *c, double dt)
{
    // N_sub = max(1, ceil(dt c_hat / (CFL dx))), with a 1e-12 relative
    // slack so that dt = N CFL dx / c_hat gives exactly N.
    const double ratio = dt * c->pc.c_hat / (c->pc.cfl * c->pc.dx);
    const int n = (int)ceil(ratio * (1.0 - 1e-12));
    return n < 1 ? 1 : n;
}

}  // namespace

// =================================================================================================
// C ABI
// =================================================================================================
extern "C" {

const char *qk_version(void) { return "quokka-b200 0.1 (sm_100a, fp64, -fmad=false)"; }

int qk_init(int nx, int ny, int nz, double dx, double gamma, double c_hat, double c, int boundary, qk_ctx **out)
{
    if (!out) return QK_EINVAL;
    *out = nullptr;
    if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0.0) || !(gamma > 1.0) || c_hat < 0.0 || c < 0.0) return QK_EINVAL;
    if (boundary < QK_BC_PERIODIC || boundary > QK_BC_FIXED) return QK_EINVAL;
    if ((long long)(nx + 2 * NG) * (ny + 2 * NG) * (nz + 2 * NG) > 2000000000LL) return QK_EINVAL;
    if (ny + 4 > 65535 || nz + 4 > 65535) return QK_EINVAL;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return QK_ECUDA; }
    qk_ctx *x = new (std::nothrow) qk_ctx();
    if (!x) return QK_ENOMEM;
    x->g = make_geom(nx, ny, nz);
    x->pc.dx = dx; x->pc.gamma = gamma; x->pc.c_hat = c_hat; x->pc.c = c;
    x->pc.a_rad = 1.0; x->pc.kB_mu = 1.0; x->pc.eos_alpha = 0.0;
    x->pc.opac_kP0 = 0.0; x->pc.opac_kR0 = 0.0; x->pc.opac_rho0 = 0.0; x->pc.opac_exp = 0; x->pc.cfl = 0.3; x->pc.newton_tol = 1e-10;
    x->pc.newton_maxit = 400; x->pc.nsub_max = 10; x->pc.flags = QK_FLAG_TAU_CORR; x->pc.bc = boundary;
    x->stream = nullptr; x->device = dev; x->base = nullptr; x->bytes = 0; x->owns = false; x->ready = false;
    x->path = QK_PATH_SWEEP; x->w_cur = 0; x->s_cur = 0; x->w_valid = false; x->s_valid = false; x->smax_valid = false; x->has_source = false; x->has_fixed = boundary == QK_BC_FIXED;
    for (int f = 0; f < 6; ++f) x->fb.t[f] = boundary;
    x->ext_faces = 0; x->halo_fn = nullptr; x->halo_user = nullptr; x->pending.n = 0; x->in_halo_cb = false;
    x->launches = 0; x->last_nsub = 0; x->profiling = false;
    *out = x;
    return QK_OK;
}

int qk_free(qk_ctx *c)
{
    if (!c) return QK_EINVAL;
    if (c->ready) cudaStreamSynchronize(c->stream);
    for (auto &s : c->spans) { cudaEventDestroy(s.a); cudaEventDestroy(s.b); }
    for (auto e : c->pool) cudaEventDestroy(e);
    if (c->owns && c->base) cudaFree(c->base);
    delete c;
    return QK_OK;
}

size_t qk_state_bytes(int nx, int ny, int nz)
{
    if (nx < 1 || ny < 1 || nz < 1) return 0;
    return total_bytes(make_geom(nx, ny, nz));
}

int qk_bind_storage(qk_ctx *c, void *dev_ptr, size_t bytes)
{
    if (!c || !dev_ptr || c->ready) return QK_EINVAL;
    if (bytes < total_bytes(c->g) || ((size_t)dev_ptr & 255) != 0 || !is_device_ptr(dev_ptr)) return QK_EINVAL;
    c->base = (char *)dev_ptr;
    c->bytes = total_bytes(c->g);
    c->owns = false;
    return QK_OK;
}

int qk_set_stream(qk_ctx *c, void *cuda_stream)
{
    if (!c) return QK_EINVAL;
    c->stream = (cudaStream_t)cuda_stream;
    return QK_OK;
}

int qk_set_constants(qk_ctx *c, double a_rad, double kB_over_mu_mH)
{
    if (!c || !(a_rad >= 0.0) || !(kB_over_mu_mH > 0.0)) return QK_EINVAL;
    c->pc.a_rad = a_rad; c->pc.kB_mu = kB_over_mu_mH;
    return QK_OK;
}

int qk_set_face_boundaries(qk_ctx *c, const int *bc6)
{
    if (!c || !bc6) return QK_EINVAL;
    for (int f = 0; f < 6; ++f)
        if (bc6[f] < QK_BC_PERIODIC || bc6[f] > QK_BC_FIXED) return QK_EINVAL;
    for (int a = 0; a < 3; ++a)
        if ((bc6[2 * a] == QK_BC_PERIODIC) != (bc6[2 * a + 1] == QK_BC_PERIODIC)) return QK_EINVAL;
    c->has_fixed = false;
    for (int f = 0; f < 6; ++f) { c->fb.t[f] = bc6[f]; c->has_fixed = c->has_fixed || bc6[f] == QK_BC_FIXED; }
    c->w_valid = false; c->s_valid = false;
    return QK_OK;
}

int qk_set_opacity_law(qk_ctx *c, double kappaP0, double kappaR0, double rho0, int exponent)
{
    if (!c || !(kappaP0 >= 0.0) || !(kappaR0 >= 0.0) || !(rho0 >= 0.0) || exponent < -4 || exponent > 4) return QK_EINVAL;
    c->pc.opac_kP0 = kappaP0; c->pc.opac_kR0 = kappaR0; c->pc.opac_rho0 = rho0; c->pc.opac_exp = exponent;
    return QK_OK;
}

int qk_set_eos(qk_ctx *c, int eos, double alpha)
{
    if (!c || (eos != QK_EOS_IDEAL && eos != QK_EOS_ALPHA_T3) || (eos == QK_EOS_ALPHA_T3 && !(alpha > 0.0))) return QK_EINVAL;
    c->pc.eos_alpha = eos == QK_EOS_ALPHA_T3 ? alpha : 0.0;
    return QK_OK;
}

int qk_set_params(qk_ctx *c, double cfl, double newton_tol, int newton_maxit, int nsub_max, unsigned flags)
{
    if (!c || !(cfl > 0.0) || !(newton_tol > 0.0) || newton_maxit < 1 || nsub_max < 1) return QK_EINVAL;
    if ((flags & QK_FLAG_EDDINGTON) && (flags & QK_FLAG_MINERBO)) return QK_EINVAL;
    c->pc.cfl = cfl; c->pc.newton_tol = newton_tol; c->pc.newton_maxit = newton_maxit;
    c->pc.nsub_max = nsub_max; c->pc.flags = flags;
    return QK_OK;
}

int qk_set_path(qk_ctx *c, int path)
{
    if (!c || path < QK_PATH_FUSED || path > QK_PATH_SWEEP) return QK_EINVAL;
    c->path = path;
    c->w_valid = false; c->s_valid = false;
    return QK_OK;
}

int qk_set_state(qk_ctx *c, int field, const double *interior)
{
    if (!c || field < 0 || field >= QK_NFIELDS || !interior) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    if (field == QK_SRC) c->has_source = true;
    else { c->w_valid = false; c->s_valid = false; c->smax_valid = false; }
    rc = copy_interior(c, c->state[field], const_cast<double *>(interior), true);
    // pageable host memory may be reused by the caller as soon as we return
    if (rc == QK_OK && !is_device_ptr(interior) && cudaStreamSynchronize(c->stream) != cudaSuccess) rc = QK_ECUDA;
    return rc;
}

int qk_get_state(qk_ctx *c, int field, double *interior)
{
    if (!c || field < 0 || field >= QK_NFIELDS || !interior) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    rc = copy_interior(c, c->state[field], interior, false);
    if (rc == QK_OK && cudaStreamSynchronize(c->stream) != cudaSuccess) rc = QK_ECUDA;
    return rc;
}

int qk_set_raw(qk_ctx *c, int field, const double *with_ghosts)
{
    if (!c || field < 0 || field >= QK_NFIELDS || !with_ghosts) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    if (field == QK_SRC) c->has_source = true;
    else { c->w_valid = false; c->s_valid = false; c->smax_valid = false; }
    if (cudaMemcpyAsync(c->state[field], with_ghosts, (size_t)c->g.ntot * sizeof(double), cudaMemcpyDefault,
                        c->stream) != cudaSuccess) return QK_ECUDA;
    return cudaStreamSynchronize(c->stream) == cudaSuccess ? QK_OK : QK_ECUDA;
}

int qk_get_raw(qk_ctx *c, int field, double *with_ghosts)
{
    if (!c || field < 0 || field >= QK_NFIELDS || !with_ghosts) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    if (cudaMemcpyAsync(with_ghosts, c->state[field], (size_t)c->g.ntot * sizeof(double), cudaMemcpyDefault,
                        c->stream) != cudaSuccess) return QK_ECUDA;
    return cudaStreamSynchronize(c->stream) == cudaSuccess ? QK_OK : QK_ECUDA;
}

int qk_fill_boundary(qk_ctx *c, int which)
{
    if (!c || (which & ~QK_FILL_ALL)) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    double *list[QK_NFIELDS];
    signed char comps[QK_NFIELDS];
    static const signed char comp_of[QK_NFIELDS] = {-1, 0, 1, 2, -1, -1, 0, 1, 2, -1, -1, -1};
    int n = 0;
    auto add = [&](int f) { list[n] = c->state[f]; comps[n] = comp_of[f]; ++n; };
    if (which & QK_FILL_HYDRO) for (int f = QK_RHO; f <= QK_E; ++f) add(f);
    if (which & QK_FILL_RAD) for (int f = QK_ER; f <= QK_FZ; ++f) add(f);
    if (which & QK_FILL_OPACITY) for (int f = QK_KAPPA_P; f <= QK_KAPPA_R; ++f) add(f);
    fill_fields(c, list, n, comps);
    return check_launch();
}

int qk_set_halo_exchange(qk_ctx *c, unsigned faces, qk_halo_fn fn, void *user)
{
    if (!c || (faces & ~(unsigned)(QK_FACE_ZLO | QK_FACE_ZHI))) return QK_EINVAL;
    if (faces && fn && c->g.nz < NG) return QK_EINVAL;
    c->ext_faces = fn ? faces : 0u;
    c->halo_fn = faces ? fn : nullptr;
    c->halo_user = user;
    return QK_OK;
}

size_t qk_halo_doubles(const qk_ctx *c) { return c ? (size_t)NG * c->g.ny * c->g.nx : 0; }

static int halo_copy(qk_ctx *c, int face, double *buf, int unpack)
{
    if (!c || !buf || !c->in_halo_cb || (face != QK_FACE_ZLO && face != QK_FACE_ZHI) || !(c->ext_faces & face))
        return QK_EINVAL;
    c->launches += launch_halo_copy(c->g, face == QK_FACE_ZHI, unpack, c->pending, buf, c->stream);
    return check_launch();
}

int qk_halo_pack(qk_ctx *c, int face, double *dev_buf) { return halo_copy(c, face, dev_buf, 0); }
int qk_halo_unpack(qk_ctx *c, int face, const double *dev_buf) { return halo_copy(c, face, const_cast<double *>(dev_buf), 1); }

double qk_cfl_dt(qk_ctx *c)
{
    if (!c || ensure_storage(c) != QK_OK) return NAN;
    if (!c->smax_valid) {                // otherwise the kernel that wrote the state left its speed in the cache
        cudaMemsetAsync(c->cache, 0, sizeof(StateCache), c->stream);
        Scope s(c, K_CFL);
        s.done(launch_cfl(c->g, c->pc.gamma, ch5(&c->state[QK_RHO]), c->cache, c->stream));
        c->smax_valid = true;
    }
    unsigned long long host[2];
    if (cudaMemcpyAsync(host, c->cache, sizeof(host), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess) { cudaGetLastError(); return NAN; }
    if (host[1] != 0) return NAN;
    double smax;
    memcpy(&smax, &host[0], sizeof(double));
    double dt = c->pc.cfl * c->pc.dx / smax;                              // eq 21
    if (c->pc.c_hat > 0.0) {
        const double dtr = (double)c->pc.nsub_max * (c->pc.cfl * c->pc.dx / c->pc.c_hat);
        if (dtr < dt) dt = dtr;
    }
    return dt;
}

int qk_hydro_step(qk_ctx *c, double dt)
{
    if (!c || !(dt > 0.0)) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    reset_counters(c);
    c->last_nsub = 0;
    return do_hydro_step(c, dt);
}

int qk_hydro_step_cfl(qk_ctx *c)
{
    if (!c) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    if (c->path != QK_PATH_SWEEP) return QK_EINVAL;
    reset_counters(c);
    c->last_nsub = 0;
    if (!c->smax_valid) {
        cudaMemsetAsync(c->cache, 0, sizeof(StateCache), c->stream);
        Scope s(c, K_CFL);
        s.done(launch_cfl(c->g, c->pc.gamma, ch5(&c->state[QK_RHO]), c->cache, c->stream));
        c->smax_valid = true;
    }
    {
        Scope s(c, K_CFL);
        s.done(launch_dt_from_cache(c->cache, c->ddt, c->pc.cfl, c->pc.dx, c->pc.c_hat, c->pc.nsub_max, c->stream));
    }
    return do_hydro_step(c, 1.0, &c->ddt->dtdx);
}

int qk_last_dt(qk_ctx *c, double *dt)
{
    if (!c || !dt) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    DeviceDt h;
    if (cudaMemcpyAsync(&h, c->ddt, sizeof(h), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess) { cudaGetLastError(); return QK_ECUDA; }
    *dt = h.dt;
    return QK_OK;
}

int qk_rad_transport(qk_ctx *c, double dt)
{
    if (!c || !(dt > 0.0) || !(c->pc.c_hat > 0.0) || !(c->pc.c > 0.0)) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    reset_counters(c);
    c->last_nsub = 1;
    return do_rad_transport(c, dt);
}

int qk_exchange(qk_ctx *c, double dt)
{
    if (!c || !(dt > 0.0) || !(c->pc.c_hat > 0.0) || !(c->pc.c > 0.0)) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    reset_counters(c);
    c->last_nsub = 1;
    return do_exchange(c, dt);
}

int qk_rad_step(qk_ctx *c, double dt)
{
    if (!c || !(dt > 0.0) || !(c->pc.c_hat > 0.0) || !(c->pc.c > 0.0)) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    reset_counters(c);
    c->last_nsub = 1;
    rc = do_rad_transport(c, dt);
    if (rc) return rc;
    return do_exchange(c, dt);                 // once per subcycle (R9)
}

int qk_nsub_for(const qk_ctx *c, double dt)
{
    if (!c || !(c->pc.c_hat > 0.0)) return 0;
    return nsub_for(c, dt);
}

int qk_rhd_step(qk_ctx *c, double dt)
{
    if (!c || !(dt > 0.0) || !(c->pc.c_hat > 0.0) || !(c->pc.c > 0.0)) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    const int nsub = nsub_for(c, dt);
    if (nsub > c->pc.nsub_max) return QK_EINVAL;
    reset_counters(c);
    rc = do_hydro_step(c, dt);
    if (rc) return rc;
    const double dts = dt / (double)nsub;
    for (int s = 0; s < nsub; ++s) {
        rc = do_rad_transport(c, dts);
        if (rc) return rc;
        rc = do_exchange(c, dts);
        if (rc) return rc;
    }
    c->last_nsub = nsub;
    return QK_OK;
}

int qk_last_info(qk_ctx *c, qk_info *out)
{
    if (!c || !out) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    Counters h;
    StateCache sc;
    if (cudaMemcpyAsync(&h, c->ctr, sizeof(h), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
        cudaMemcpyAsync(&sc, c->cache, sizeof(sc), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess) { cudaGetLastError(); return QK_ECUDA; }
    out->nsub = c->last_nsub;
    out->newton_max_iters = h.newton_max;
    out->newton_fail_cells = h.newton_fail;
    out->newton_total_iters = h.newton_total;
    out->bad_state_cells = h.bad_state;
    out->fallback_states = h.fallback;
    out->guard_faces = h.guard;
    const bool cfl_bad = c->smax_valid && sc.cfl_bad != 0;     // set by the last qk_cfl_dt / hydro step
    out->status = h.newton_fail ? QK_ENEWTON : ((h.bad_state || cfl_bad) ? QK_ESTATE : QK_OK);
    return QK_OK;
}

long long qk_launch_count(const qk_ctx *c) { return c ? c->launches : -1; }

int qk_set_profiling(qk_ctx *c, int on)
{
    if (!c) return QK_EINVAL;
    c->profiling = on != 0;
    return QK_OK;
}

int qk_kernel_class_count(void) { return K_NCLASS; }

const char *qk_kernel_class_name(int cls)
{
    static const char *names[K_NCLASS] = {"fill_boundary", "cfl", "prim", "flatten", "hydro_flux", "hydro_update",
                                          "hydro_stage", "rad_prim", "rad_flux", "rad_update", "rad_stage", "exchange",
                                          "hydro_sweep_x", "hydro_sweep_y", "hydro_sweep_z", "rad_sweep_x",
                                          "rad_sweep_y", "rad_sweep_z"};
    return (cls >= 0 && cls < K_NCLASS) ? names[cls] : "";
}

int qk_kernel_times(qk_ctx *c, double *ms, long long *count)
{
    if (!c || !ms || !count) return QK_EINVAL;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return QK_ECUDA;
    for (int k = 0; k < K_NCLASS; ++k) { ms[k] = 0.0; count[k] = 0; }
    for (auto &s : c->spans) {
        float t = 0.f;
        if (cudaEventElapsedTime(&t, s.a, s.b) == cudaSuccess) { ms[s.cls] += (double)t; count[s.cls] += 1; }
        c->pool.push_back(s.a);
        c->pool.push_back(s.b);
    }
    c->spans.clear();
    return QK_OK;
}

}  // extern "C"

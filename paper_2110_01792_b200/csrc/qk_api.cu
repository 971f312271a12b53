// qk_api.cu -- the C ABI of include/qk.h: context, device storage layout, step drivers.
//
// Storage (one allocation, caller- or library-owned), all fp64 SoA, each array padded to a
// multiple of 32 doubles so every field starts 256-byte aligned:
//   [ 12 state fields | 5 RK stage fields | chi and its 3 directional parts | 5 flux-difference accumulators D |
//     2 x 5 primitive fields W (ping-pong between RK stages) | 2 x 4 radiation fields S = (E_r, f) | counters ]
// Drivers follow the operator-split cycle of PAPER.md:112: hydro step (SSP-RK2),
// then N_sub x (radiation transport RK2, exchange).
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <new>

#include <cuda.h>          // types of the two driver entry points fetched at run time (no libcuda link)
#include <unistd.h>

#include "qk_internal.h"

using namespace qk;

namespace {

constexpr int N_STAGE = 5;          // U^(1) (hydro) / first 4 reused for radiation
constexpr int N_ACC = 5;            // D = dF_x + dF_y per conserved variable (first 4 reused for radiation)
constexpr int N_RECON = 18;         // W_A (5), W_B (5), S_A (4), S_B (4)
constexpr int RC_WA = 0, RC_WB = 5, RC_SA = 10, RC_SB = 14;
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
    double *chi3[3];       // directional flattening coefficients
    int chi_path;          // qk_set_flatten_path
    double *acc[N_ACC];
    double *recon[N_RECON];
    Counters *ctr;
    StateCache *cache;
    DeviceDt *ddt;         // device-resident timestep of qk_hydro_step_cfl / qk_rhd_step_cfl
    // which W / S set holds the reconstruction variables of the current state (interior cells; written by the kernel
    // that produced the state), and whether it / the cached CFL speed still describe the state
    int w_cur, s_cur;
    bool w_valid, s_valid, smax_valid;
    FaceBc fb;             // boundary type of each face (qk_init sets all six alike)
    bool has_fixed;        // some face is QK_BC_FIXED: the ghost cells beyond it hold caller-supplied values
    bool has_source;       // QK_SRC was set: the exchange reads it (otherwise S = 0 and the field is never touched)
    // z-slab decomposition: inter-rank faces, the caller's halo mover, and the field list of the fill in progress
    unsigned ext_faces;
    qk_halo_fn halo_fn;
    void *halo_user;
    FillList pending;
    bool in_halo_cb;
    bool halo_failed;      // a halo callback reported an error: later step calls return QK_EINVAL
    // peer-mapped exchange (qk_set_halo_peers): the neighbours' storage, mapped into this process
    struct Peer { char *base; Geom g; size_t fs; unsigned long long *flag; void *ipc_ptr; } peer[2];   // lo, hi
    bool peers_on;
    unsigned long long epoch;            // number of ghost fills so far: the value the arrival counters must reach
    unsigned long long *arrive;          // [2] in this context's counter block: written by the lo / hi neighbour
    cudaStream_t side;                   // stream of the pushes
    cudaEvent_t ev_main, ev_side;
    bool fill_open;                      // between fill_begin and fill_end
    // host copies: copy stream + events of the pipelined qk_set_state_all / qk_get_state_all
    cudaStream_t copy_stream;
    cudaEvent_t ev_copy, ev_compute;
    long long launches;
    int last_nsub;
    // replayable step (qk_graph_capture): the instantiated CUDA graph of one step and everything host-side that its
    // launch sequence and kernel arguments were derived from -- a launch with another signature is refused
    struct StepGraph {
        cudaGraphExec_t exec;
        int kind, nsub, launches;
        PhysConsts pc; FaceBc fb; bool has_fixed, has_source; int chi_path; cudaStream_t stream; void *base;
    } graph;
    // per-kernel-class event timing
    bool profiling;
    struct Span { int cls; cudaEvent_t a, b; };
    std::vector<Span> spans;
    std::vector<cudaEvent_t> pool;
};

namespace {

size_t total_bytes(const Geom &g)
{
    const size_t nf = QK_NFIELDS + N_STAGE + 4 + N_ACC + N_RECON;
    return nf * field_stride(g) * sizeof(double) + COUNTER_BYTES;
}

int carve(qk_ctx *c)
{
    const size_t fs = field_stride(c->g);
    double *p = (double *)c->base;
    for (int f = 0; f < QK_NFIELDS; ++f) { c->state[f] = p; p += fs; }
    for (int f = 0; f < N_STAGE; ++f) { c->stage[f] = p; p += fs; }
    c->chi = p; p += fs;
    for (int f = 0; f < 3; ++f) { c->chi3[f] = p; p += fs; }
    for (int f = 0; f < N_ACC; ++f) { c->acc[f] = p; p += fs; }
    for (int f = 0; f < N_RECON; ++f) { c->recon[f] = p; p += fs; }
    c->ctr = (Counters *)p;
    c->cache = (StateCache *)((char *)p + 128);
    c->arrive = (unsigned long long *)((char *)p + 160);
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

// copy between a dense interior array (planes [k0, k1) of it) and the ghosted field, on stream `st`
int copy_interior(qk_ctx *c, double *field, double *dense, bool to_field, cudaStream_t st, int k0 = 0, int k1 = -1)
{
    const Geom &g = c->g;
    if (k1 < 0) k1 = g.nz;
    cudaMemcpy3DParms p;
    memset(&p, 0, sizeof(p));
    cudaPitchedPtr fptr = make_cudaPitchedPtr(field, (size_t)g.px * sizeof(double), g.px, g.py);
    cudaPitchedPtr dptr = make_cudaPitchedPtr(dense, (size_t)g.nx * sizeof(double), g.nx, g.ny);
    const cudaPos fpos = make_cudaPos((size_t)NG * sizeof(double), NG, NG + k0);
    const cudaPos dpos = make_cudaPos(0, 0, k0);
    if (to_field) { p.srcPtr = dptr; p.srcPos = dpos; p.dstPtr = fptr; p.dstPos = fpos; }
    else          { p.srcPtr = fptr; p.srcPos = fpos; p.dstPtr = dptr; p.dstPos = dpos; }
    p.extent = make_cudaExtent((size_t)g.nx * sizeof(double), g.ny, k1 - k0);
    p.kind = cudaMemcpyDefault;
    return cudaMemcpy3DAsync(&p, st) == cudaSuccess ? QK_OK : QK_ECUDA;
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

// stream memory operation of the driver (cuStreamWaitValue64), fetched once; nullptr: not available (then
// qk_set_halo_peers refuses: a kernel that polls a counter another rank writes must never be launched)
typedef CUresult (*wait_value_fn)(CUstream, CUdeviceptr, cuuint64_t, unsigned int);
wait_value_fn stream_wait_value()
{
    static bool looked = false;
    static wait_value_fn fn = nullptr;
    if (!looked) {
        looked = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuStreamWaitValue64", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess) fn = (wait_value_fn)p;
        else cudaGetLastError();
    }
    return fn;
}

// Every list the drivers fill is (scalar, x, y, z component, scalars ...): U, W, R, S, optionally followed by rho
// and kappa_R; qk_fill_boundary passes the components of its own list.  fixed_src: see FillList.
//
// fill_begin starts the ghost fill of a field list, fill_end completes it; kernels that read no z ghost plane may be
// launched in between.  Single box / callback exchange: everything happens in fill_begin.  Peer-mapped exchange:
//   fill_begin : side stream (after the main stream's work so far): push my boundary planes into the neighbours'
//                ghost planes, then raise their arrival counters to this fill's epoch;  main stream: fill every ghost
//                cell that does not depend on the neighbours (x / y images of the interior planes, physical z faces);
//   fill_end   : main stream waits until my own counters reach the epoch (a stream memory operation: no kernel spins,
//                no host wait), then fills the x / y images of the received planes.
// So the transfer overlaps whatever the caller launches between the two.
int fill_begin(qk_ctx *c, double *const *fields, int n, const signed char *comps = nullptr,
               double *const *fixed_src = nullptr)
{
    FillList fl;
    fl.n = n;
    for (int i = 0; i < n; ++i) {
        fl.f[i] = fields[i];
        fl.fixed_src[i] = (fixed_src && c->has_fixed) ? fixed_src[i] : nullptr;
        fl.comp[i] = comps ? comps[i] : (signed char)((i >= 1 && i <= 3) ? i - 1 : -1);
    }
    c->pending = fl;
    c->fill_open = true;
    Scope s(c, K_FILL);
    if (c->peers_on) {
        ++c->epoch;
        int nl = 0;
        if (cudaEventRecord(c->ev_main, c->stream) != cudaSuccess || cudaStreamWaitEvent(c->side, c->ev_main, 0) != cudaSuccess)
            return QK_ECUDA;
        for (int side = 0; side < 2; ++side) {
            if (!(c->ext_faces & (side ? QK_FACE_ZHI : QK_FACE_ZLO))) continue;
            const qk_ctx::Peer &p = c->peer[side];
            PeerList dst;
            const size_t my_fs = field_stride(c->g);
            for (int i = 0; i < n; ++i) {
                const size_t slot = (size_t)(fl.f[i] - (double *)c->base) / my_fs;      // same slot in the neighbour's layout
                dst.f[i] = (double *)p.base + slot * p.fs;
            }
            nl += launch_halo_push(c->g, p.g, side, fl, dst, p.flag, c->epoch, c->side);
        }
        cudaEventRecord(c->ev_side, c->side);
        nl += launch_fill(c->g, c->fb, c->ext_faces, 1, fl, c->stream);
        s.done(nl);
        return QK_OK;
    }
    if (c->ext_faces && c->halo_fn) {      // neighbours' planes first, then the x / y images of everything
        c->in_halo_cb = true;
        const int hrc = c->halo_fn(c->halo_user, n);
        c->in_halo_cb = false;
        if (hrc != 0) { c->halo_failed = true; c->fill_open = false; s.done(0); return QK_EINVAL; }
    }
    s.done(launch_fill(c->g, c->fb, c->ext_faces, 0, fl, c->stream));
    return QK_OK;
}

int fill_end(qk_ctx *c)
{
    if (!c->fill_open) return QK_OK;
    c->fill_open = false;
    if (!c->peers_on) return QK_OK;
    Scope s(c, K_HALO);
    int nl = 0;
    for (int side = 0; side < 2; ++side) {
        if (!(c->ext_faces & (side ? QK_FACE_ZHI : QK_FACE_ZLO))) continue;
        if (stream_wait_value()((CUstream)c->stream, (CUdeviceptr)(c->arrive + side), (cuuint64_t)c->epoch, 0u /* GEQ */) !=
            CUDA_SUCCESS) { c->halo_failed = true; return QK_ECUDA; }
    }
    nl += launch_fill(c->g, c->fb, c->ext_faces, 2, c->pending, c->stream);
    // the planes just pushed may be overwritten by what follows only once the push has read them
    cudaStreamWaitEvent(c->stream, c->ev_side, 0);
    s.done(nl);
    return QK_OK;
}

int fill_fields(qk_ctx *c, double *const *fields, int n, const signed char *comps = nullptr,
                double *const *fixed_src = nullptr)
{
    const int rc = fill_begin(c, fields, n, comps, fixed_src);
    return rc ? rc : fill_end(c);
}

// ---- hydro: SSP-RK2 ------------------------------------------------------------------
// stage 1:  U1 = Un - (dt/dx) div F(Un)            -> stage buffers
// stage 2:  Un+1 = 0.5 Un + 0.5 (U1 - (dt/dx) div F(U1))   -> state (each cell reads only its own Un)
// One stage.  W_in holds the primitives of U for the interior cells when `w_ready` (left there by the kernel that
// produced U): the ghost fill then runs on W -- periodic / outflow / mirror images commute with the pointwise cons ->
// prim map, so the bits are those of prim(ghost-filled U).  Otherwise (fresh state, or Dirichlet faces whose ghost
// cells hold caller-supplied conserved values) U is ghost-filled and W computed for every cell.  Then the flattening
// coefficient, x sweep (D = dFx), y sweep (D += dFy), z sweep (RK update into `out`, primitives of the new cells into
// W_out; after the last stage also the CFL speed of the new state).
int hydro_stage(qk_ctx *c, double dtdx, int stage, double *const *U, double *const *U0, double *const *out,
                double *const *W, double *const *Wout, bool w_ready, const double *dtdx_dev)
{
    const Geom &g = c->g;
    const int nz = g.nz;
    auto chi = [&](int d0, int d1, int m0, int m1) {
        Scope s(c, K_FLATTEN);
        s.done(launch_chi(g, c->pc.gamma, ch5(W), c->chi3[0], c->chi3[1], c->chi3[2], c->chi, d0, d1, m0, m1, c->chi_path, c->stream));
    };
    // the density is its own primitive: the sweeps read it from the stage's state U (ghost-filled here either way), so
    // the kernel that produces a state stores four primitives, not five
    double *const Wv[5] = {U[0], W[1], W[2], W[3], W[4]};
    auto sweep = [&](int d, int k0, int k1) {
        Scope s(c, K_HYDRO_X + d);
        s.done(launch_hydro_sweeps(g, c->pc.gamma, c->pc.flags, dtdx, stage, ch5(Wv), c->chi, h5(c->acc), ch5(U), ch5(U0), h5(out),
                                   h5(Wout), c->ctr, c->cache, c->stream, 1 << d, dtdx_dev, k0, k1));
    };
    int rc;
    const bool cached = w_ready && !c->has_fixed;
    if (cached) {
        rc = fill_begin(c, Wv, 5);
        if (rc) return rc;
    } else {
        rc = fill_fields(c, U, 5, nullptr, stage == 1 ? U0 : nullptr);
        if (rc) return rc;
        Scope s(c, K_PRIM);
        s.done(launch_prim(g, c->pc.gamma, ch5(U), h5(W), c->ctr, c->stream));
    }
    if (c->fill_open && c->peers_on && nz >= 8) {
        // while the neighbours' planes travel: everything that reads no z ghost plane.  chi~_z of plane k reads P at
        // k +- 2, chi of plane k reads chi~ at k +- 1, the x and y sweeps of plane k read chi and W of that plane only.
        chi(2, nz - 2, 3, nz - 3);
        sweep(0, 3, nz - 3);
        sweep(1, 3, nz - 3);
        rc = fill_end(c);
        if (rc) return rc;
        chi(-2, 2, -1, 3);
        chi(nz - 2, nz + 2, nz - 3, nz + 1);
        for (int d = 0; d < 2; ++d) { sweep(d, 0, 3); sweep(d, nz - 3, nz); }
    } else {
        rc = fill_end(c);
        if (rc) return rc;
        chi(-2, nz + 2, -1, nz + 1);
        sweep(0, 0, nz);
        sweep(1, 0, nz);
    }
    sweep(2, 0, nz);
    return QK_OK;
}

int do_hydro_step(qk_ctx *c, double dt, const double *dtdx_dev = nullptr)
{
    if (c->halo_failed) return QK_EINVAL;
    const double dtdx = dt / c->pc.dx;
    double *const *Un = &c->state[QK_RHO];
    double *const *U1 = &c->stage[0];
    double *const *W0 = &c->recon[c->w_cur ? RC_WB : RC_WA];
    double *const *W1 = &c->recon[c->w_cur ? RC_WA : RC_WB];
    int rc = hydro_stage(c, dtdx, 0, Un, Un, U1, W0, W1, c->w_valid, dtdx_dev);
    if (rc) return rc;
    cudaMemsetAsync(c->cache, 0, sizeof(StateCache), c->stream);
    rc = hydro_stage(c, dtdx, 1, U1, Un, Un, W1, W0, true, dtdx_dev);
    if (rc) return rc;
    c->w_valid = true;                   // W0 = primitives of the new state, cache = its CFL speed
    c->smax_valid = true;
    return check_launch();
}

// ---- radiation transport: same SSP-RK2 -----------------------------------------------------
int rad_stage(qk_ctx *c, double dtdx, int stage, double *const *R, double *const *R0, double *const *out,
              double *const *S, double *const *Sout, bool s_ready, const double *dtdx_dev)
{
    // rho and kappa_R ghosts feed tau_face at the domain faces (first stage of a transport step only)
    const bool cached = s_ready && !c->has_fixed;
    const int nz = c->g.nz;
    double *list[6];
    int n = 0;
    // E_r is its own reconstruction variable: read from the stage's state R (ghost-filled here either way)
    double *const Sv[4] = {R[0], S[1], S[2], S[3]};
    double *const *src = cached ? Sv : R;
    for (int f = 0; f < 4; ++f) list[n++] = src[f];
    if (stage == 0) { list[n++] = c->state[QK_RHO]; list[n++] = c->state[QK_KAPPA_R]; }
    int rc = fill_begin(c, list, n, nullptr, (!cached && stage == 1) ? R0 : nullptr);
    if (rc) return rc;
    auto sweep = [&](int d) {
        Scope s(c, K_RAD_X + d);
        s.done(launch_rad_sweeps(c->g, c->pc, dtdx, stage, cr4(Sv), c->state[QK_RHO], c->state[QK_KAPPA_R], r4(c->acc), cr4(R),
                                 cr4(R0), r4(out), r4(Sout), c->ctr, c->stream, 1 << d, dtdx_dev, 0, nz));
    };
    if (cached) {        // the x and y sweeps read no z ghost plane: they run while the neighbours' planes travel
        sweep(0);
        sweep(1);
        rc = fill_end(c);
        if (rc) return rc;
    } else {
        rc = fill_end(c);
        if (rc) return rc;
        { Scope s(c, K_PRIM); s.done(launch_rad_prim(c->g, c->pc.c, cr4(R), r4(S), c->ctr, c->stream)); }
        sweep(0);
        sweep(1);
    }
    sweep(2);
    return QK_OK;
}

int do_rad_transport(qk_ctx *c, double dt, const double *dtdx_dev = nullptr)
{
    if (c->halo_failed) return QK_EINVAL;
    if (c->pc.opac_rho0 > 0.0) {         // opacities follow the density (and temperature) the last update left (X14)
        Scope s(c, K_OPACITY);
        s.done(launch_opacity_law(c->g, c->pc, ch5(&c->state[QK_RHO]), c->state[QK_KAPPA_P], c->state[QK_KAPPA_R], c->stream));
    }
    const double dtdx = dt / c->pc.dx;
    double *const *Rn = &c->state[QK_ER];
    double *const *R1 = &c->stage[0];
    double *const *S0 = &c->recon[c->s_cur ? RC_SB : RC_SA];
    double *const *S1 = &c->recon[c->s_cur ? RC_SA : RC_SB];
    int rc = rad_stage(c, dtdx, 0, Rn, Rn, R1, S0, S1, c->s_valid, dtdx_dev);
    if (rc) return rc;
    rc = rad_stage(c, dtdx, 1, R1, Rn, Rn, S1, S0, true, dtdx_dev);
    if (rc) return rc;
    c->s_valid = true;
    return check_launch();
}

int do_exchange(qk_ctx *c, double dt, const double *dt_dev = nullptr)
{
    double *const *s = c->state;
    // the exchange rewrites rho v, E, E_r, F_r: it also refreshes what the next stages read and the CFL speed
    Hydro5 W = h5(&c->recon[c->w_cur ? RC_WB : RC_WA]);
    Rad4p S = r4(&c->recon[c->s_cur ? RC_SB : RC_SA]);
    if (c->has_fixed) { W = Hydro5{nullptr, nullptr, nullptr, nullptr, nullptr}; S = Rad4p{nullptr, nullptr, nullptr, nullptr}; }
    cudaMemsetAsync(c->cache, 0, sizeof(StateCache), c->stream);
    Scope sc(c, K_EXCHANGE);
    sc.done(launch_exchange(c->g, c->pc, dt, dt_dev, s[QK_RHO], s[QK_MX], s[QK_MY], s[QK_MZ], s[QK_E], s[QK_ER], s[QK_FX],
                            s[QK_FY], s[QK_FZ], s[QK_KAPPA_P], s[QK_KAPPA_R], c->has_source ? s[QK_SRC] : nullptr, W, S, c->ctr,
                            c->cache, c->stream));
    c->w_valid = !c->has_fixed;
    c->s_valid = !c->has_fixed;
    c->smax_valid = true;
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

// the caller overwrote a state field: what the kernels left next to the state no longer describes it
void invalidate(qk_ctx *c, int field)
{
    if (field <= QK_E) { c->w_valid = false; c->smax_valid = false; }
    if (field >= QK_ER && field <= QK_FZ) c->s_valid = false;
}

// make sure the cached CFL speed describes the current state
void ensure_speed(qk_ctx *c)
{
    if (c->smax_valid) return;
    cudaMemsetAsync(c->cache, 0, sizeof(StateCache), c->stream);
    Scope s(c, K_CFL);
    s.done(launch_cfl(c->g, c->pc.gamma, ch5(&c->state[QK_RHO]), c->cache, c->stream));
    c->smax_valid = true;
}

}  // namespace

// =================================================================================================
// C ABI
// =================================================================================================
extern "C" {

const char *qk_version(void) { return "quokka-b200 0.4 (sm_100a, fp64, -fmad=false)"; }

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
    x->pc.opac_kP0 = 0.0; x->pc.opac_kR0 = 0.0; x->pc.opac_rho0 = 0.0; x->pc.opac_exp = 0;
    x->pc.opac_texp2 = 0; x->pc.opac_T0 = 1.0;
    x->pc.cfl = 0.3; x->pc.newton_tol = 1e-10; x->pc.newton_maxit = 400; x->pc.nsub_max = 10;
    x->pc.flags = 0;                     // plain HLL: the optical-depth correction is opt-in (R6)
    x->pc.bc = boundary;
    x->stream = nullptr; x->device = dev; x->base = nullptr; x->bytes = 0; x->owns = false; x->ready = false;
    x->chi_path = 0;
    x->w_cur = 0; x->s_cur = 0; x->w_valid = false; x->s_valid = false; x->smax_valid = false; x->has_source = false; x->has_fixed = boundary == QK_BC_FIXED;
    for (int f = 0; f < 6; ++f) x->fb.t[f] = boundary;
    x->ext_faces = 0; x->halo_fn = nullptr; x->halo_user = nullptr; x->pending.n = 0; x->in_halo_cb = false;
    x->halo_failed = false; x->peers_on = false; x->epoch = 0; x->arrive = nullptr; x->side = nullptr;
    x->ev_main = nullptr; x->ev_side = nullptr; x->fill_open = false;
    for (int p = 0; p < 2; ++p) { x->peer[p].base = nullptr; x->peer[p].flag = nullptr; x->peer[p].ipc_ptr = nullptr; x->peer[p].fs = 0; }
    x->copy_stream = nullptr; x->ev_copy = nullptr; x->ev_compute = nullptr;
    x->launches = 0; x->last_nsub = 0; x->profiling = false;
    x->graph.exec = nullptr;
    *out = x;
    return QK_OK;
}

int qk_free(qk_ctx *c)
{
    if (!c) return QK_EINVAL;
    if (c->ready) cudaStreamSynchronize(c->stream);
    for (auto &s : c->spans) { cudaEventDestroy(s.a); cudaEventDestroy(s.b); }
    for (auto e : c->pool) cudaEventDestroy(e);
    if (c->copy_stream) { cudaStreamSynchronize(c->copy_stream); cudaStreamDestroy(c->copy_stream); }
    if (c->ev_copy) cudaEventDestroy(c->ev_copy);
    if (c->ev_compute) cudaEventDestroy(c->ev_compute);
    for (int p = 0; p < 2; ++p) if (c->peer[p].ipc_ptr) cudaIpcCloseMemHandle(c->peer[p].ipc_ptr);
    if (c->side) { cudaStreamSynchronize(c->side); cudaStreamDestroy(c->side); }
    if (c->ev_main) cudaEventDestroy(c->ev_main);
    if (c->ev_side) cudaEventDestroy(c->ev_side);
    if (c->graph.exec) cudaGraphExecDestroy(c->graph.exec);
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
    return qk_set_opacity_law_T(c, kappaP0, kappaR0, rho0, exponent, 1.0, 0);
}

int qk_set_opacity_law_T(qk_ctx *c, double kappaP0, double kappaR0, double rho0, int exponent, double T0, int texp2)
{
    if (!c || !(kappaP0 >= 0.0) || !(kappaR0 >= 0.0) || !(rho0 >= 0.0) || exponent < -4 || exponent > 4) return QK_EINVAL;
    if (!(T0 > 0.0) || texp2 < -16 || texp2 > 16) return QK_EINVAL;
    c->pc.opac_kP0 = kappaP0; c->pc.opac_kR0 = kappaR0; c->pc.opac_rho0 = rho0; c->pc.opac_exp = exponent;
    c->pc.opac_T0 = T0; c->pc.opac_texp2 = texp2;
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

int qk_set_state(qk_ctx *c, int field, const double *interior)
{
    if (!c || field < 0 || field >= QK_NFIELDS || !interior) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    if (field == QK_SRC) c->has_source = true;
    else invalidate(c, field);
    rc = copy_interior(c, c->state[field], const_cast<double *>(interior), true, c->stream);
    // pageable host memory may be reused by the caller as soon as we return
    if (rc == QK_OK && !is_device_ptr(interior) && cudaStreamSynchronize(c->stream) != cudaSuccess) rc = QK_ECUDA;
    return rc;
}

int qk_get_state(qk_ctx *c, int field, double *interior)
{
    if (!c || field < 0 || field >= QK_NFIELDS || !interior) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    rc = copy_interior(c, c->state[field], interior, false, c->stream);
    if (rc == QK_OK && cudaStreamSynchronize(c->stream) != cudaSuccess) rc = QK_ECUDA;
    return rc;
}

// ---- pipelined host <-> device transfers -------------------------------------------------------------
// All fields of one call go out as one cudaMemcpy3DAsync each on the context's copy stream, ordered against the
// compute stream by events only (no host synchronisation): with pinned host memory and two contexts the upload of
// the next box, the step of this one and the download of the previous one overlap (PCIe is full duplex).
static int copy_setup(qk_ctx *c)
{
    if (c->copy_stream) return QK_OK;
    if (cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_copy, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_compute, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); return QK_ECUDA; }
    return QK_OK;
}

int qk_set_state_all(qk_ctx *c, int n, const int *fields, const double *const *interiors)
{
    if (!c || n < 1 || n > QK_NFIELDS || !fields || !interiors) return QK_EINVAL;
    for (int m = 0; m < n; ++m)
        if (fields[m] < 0 || fields[m] >= QK_NFIELDS || !interiors[m]) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc == QK_OK) rc = copy_setup(c);
    if (rc) return rc;
    // the copies must not overtake compute work that still reads the state
    if (cudaEventRecord(c->ev_compute, c->stream) != cudaSuccess || cudaStreamWaitEvent(c->copy_stream, c->ev_compute, 0) != cudaSuccess)
        return QK_ECUDA;
    for (int m = 0; m < n; ++m) {
        if (fields[m] == QK_SRC) c->has_source = true;
        else invalidate(c, fields[m]);
        rc = copy_interior(c, c->state[fields[m]], const_cast<double *>(interiors[m]), true, c->copy_stream);
        if (rc) return rc;
    }
    if (cudaEventRecord(c->ev_copy, c->copy_stream) != cudaSuccess || cudaStreamWaitEvent(c->stream, c->ev_copy, 0) != cudaSuccess)
        return QK_ECUDA;
    return QK_OK;
}

int qk_get_state_all(qk_ctx *c, int n, const int *fields, double *const *interiors)
{
    if (!c || n < 1 || n > QK_NFIELDS || !fields || !interiors) return QK_EINVAL;
    for (int m = 0; m < n; ++m)
        if (fields[m] < 0 || fields[m] >= QK_NFIELDS || !interiors[m]) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc == QK_OK) rc = copy_setup(c);
    if (rc) return rc;
    if (cudaEventRecord(c->ev_compute, c->stream) != cudaSuccess || cudaStreamWaitEvent(c->copy_stream, c->ev_compute, 0) != cudaSuccess)
        return QK_ECUDA;
    for (int m = 0; m < n; ++m) {
        rc = copy_interior(c, c->state[fields[m]], interiors[m], false, c->copy_stream);
        if (rc) return rc;
    }
    // later compute work (the next upload is ordered by qk_set_state_all itself) must not overwrite what is being read
    if (cudaEventRecord(c->ev_copy, c->copy_stream) != cudaSuccess || cudaStreamWaitEvent(c->stream, c->ev_copy, 0) != cudaSuccess)
        return QK_ECUDA;
    return QK_OK;
}

int qk_wait_copies(qk_ctx *c)
{
    if (!c) return QK_EINVAL;
    if (!c->copy_stream) return QK_OK;
    return cudaStreamSynchronize(c->copy_stream) == cudaSuccess ? QK_OK : QK_ECUDA;
}

int qk_set_raw(qk_ctx *c, int field, const double *with_ghosts)
{
    if (!c || field < 0 || field >= QK_NFIELDS || !with_ghosts) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    if (field == QK_SRC) c->has_source = true;
    else invalidate(c, field);
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
    rc = fill_fields(c, list, n, comps);
    return rc ? rc : check_launch();
}

int qk_set_halo_exchange(qk_ctx *c, unsigned faces, qk_halo_fn fn, void *user)
{
    if (!c || (faces & ~(unsigned)(QK_FACE_ZLO | QK_FACE_ZHI))) return QK_EINVAL;
    if (faces && fn && c->g.nz < NG) return QK_EINVAL;
    c->peers_on = false;
    c->ext_faces = fn ? faces : 0u;
    c->halo_fn = faces ? fn : nullptr;
    c->halo_user = user;
    c->halo_failed = false;
    return QK_OK;
}

// ---- peer-mapped exchange --------------------------------------------------------------------------------
int qk_halo_export(qk_ctx *c, qk_halo_handle *out)
{
    if (!c || !out) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return QK_ECUDA;      // storage zeroed, counters at 0
    memset(out, 0, sizeof(*out));
    out->base = (unsigned long long)(size_t)c->base;
    out->pid = (long long)getpid();
    out->device = c->device;
    out->nx = c->g.nx; out->ny = c->g.ny; out->nz = c->g.nz;
    // the IPC handle names the whole allocation the storage lives in: remember the offset into it
    typedef CUresult (*range_fn)(CUdeviceptr *, size_t *, CUdeviceptr);
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    CUdeviceptr abase = 0;
    size_t asize = 0;
    if (cudaGetDriverEntryPoint("cuMemGetAddressRange", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess &&
        ((range_fn)p)(&abase, &asize, (CUdeviceptr)(size_t)c->base) == CUDA_SUCCESS) {
        out->offset = (unsigned long long)((size_t)c->base - (size_t)abase);
        cudaIpcMemHandle_t h;
        if (cudaIpcGetMemHandle(&h, (void *)(size_t)abase) == cudaSuccess) {
            static_assert(sizeof(h) <= sizeof(out->ipc), "qk_halo_handle.ipc too small");
            memcpy(out->ipc, &h, sizeof(h));
            out->has_ipc = 1;
        } else {
            cudaGetLastError();          // e.g. memory from a virtual-memory pool: usable inside this process only
        }
    } else {
        cudaGetLastError();
    }
    return QK_OK;
}

int qk_set_halo_peers(qk_ctx *c, const qk_halo_handle *lo, const qk_halo_handle *hi)
{
    if (!c) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    for (int p = 0; p < 2; ++p) {
        if (c->peer[p].ipc_ptr) { cudaIpcCloseMemHandle(c->peer[p].ipc_ptr); c->peer[p].ipc_ptr = nullptr; }
        c->peer[p].base = nullptr;
    }
    c->peers_on = false;
    c->ext_faces = 0;
    c->halo_fn = nullptr;
    c->halo_failed = false;
    if (!lo && !hi) return QK_OK;
    if (c->g.nz < NG || !stream_wait_value()) return QK_EINVAL;
    const qk_halo_handle *hs[2] = {lo, hi};
    for (int p = 0; p < 2; ++p) {
        const qk_halo_handle *h = hs[p];
        if (!h) continue;
        if (h->nx != c->g.nx || h->ny != c->g.ny || h->nz < NG) return QK_EINVAL;
        char *base = nullptr;
        if (h->pid == (long long)getpid()) {
            base = (char *)(size_t)h->base;                        // same address space
            if (h->device != c->device) {
                int can = 0;
                cudaDeviceCanAccessPeer(&can, c->device, h->device);
                if (!can) return QK_EINVAL;
                if (cudaDeviceEnablePeerAccess(h->device, 0) != cudaSuccess) cudaGetLastError();   // already enabled is fine
            }
        } else {
            if (!h->has_ipc) return QK_EINVAL;
            cudaIpcMemHandle_t ih;
            memcpy(&ih, h->ipc, sizeof(ih));
            void *mapped = nullptr;
            if (p == 1 && lo && c->peer[0].ipc_ptr && lo->pid == h->pid && lo->base == h->base) {
                mapped = c->peer[0].ipc_ptr;        // two ranks, periodic: both neighbours are the one peer -- one mapping, owned by peer[0]
            } else {
                if (cudaIpcOpenMemHandle(&mapped, ih, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) { cudaGetLastError(); return QK_ECUDA; }
                c->peer[p].ipc_ptr = mapped;
            }
            base = (char *)mapped + h->offset;
        }
        qk_ctx::Peer &pr = c->peer[p];
        pr.base = base;
        pr.g = make_geom(h->nx, h->ny, h->nz);
        pr.fs = field_stride(pr.g);
        // the neighbour's counter block follows its fields; I am the HIGH neighbour of my low peer: I raise its arrive[1]
        char *ctr = base + (total_bytes(pr.g) - COUNTER_BYTES);
        pr.flag = (unsigned long long *)(ctr + 160) + (p == 0 ? 1 : 0);
        c->ext_faces |= p ? QK_FACE_ZHI : QK_FACE_ZLO;
    }
    if (!c->side) {
        if (cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->ev_main, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->ev_side, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); return QK_ECUDA; }
    }
    // counters restart with the exchange: both sides of a face must (re)attach before either steps
    c->epoch = 0;
    if (cudaMemsetAsync(c->arrive, 0, 2 * sizeof(unsigned long long), c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess) return QK_ECUDA;
    c->peers_on = true;
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
    ensure_speed(c);                     // usually a no-op: the kernel that wrote the state left its speed in the cache
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

// device-resident timestep: dt of eq 21 from the cached speed, limited to nsub_limit CFL dx / c_hat, and its
// nsub-th part for the radiation substeps
static void device_dt(qk_ctx *c, int nsub_limit, int nsub)
{
    ensure_speed(c);
    Scope s(c, K_CFL);
    s.done(launch_dt_from_cache(c->cache, c->ddt, c->pc.cfl, c->pc.dx, c->pc.c_hat, nsub_limit, nsub, c->stream));
}

int qk_hydro_step_cfl(qk_ctx *c)
{
    if (!c) return QK_EINVAL;
    if (c->ext_faces) return QK_EINVAL;  // a slab's own speed is not the global one: take qk_cfl_dt, reduce over ranks, qk_hydro_step
    int rc = ensure_storage(c);
    if (rc) return rc;
    reset_counters(c);
    c->last_nsub = 0;
    device_dt(c, c->pc.nsub_max, 1);
    return do_hydro_step(c, 1.0, &c->ddt->dtdx);
}

int qk_rhd_step_cfl(qk_ctx *c, int nsub)
{
    if (!c || nsub < 1 || nsub > c->pc.nsub_max || !(c->pc.c_hat > 0.0) || !(c->pc.c > 0.0)) return QK_EINVAL;
    if (c->ext_faces) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    reset_counters(c);
    device_dt(c, nsub, nsub);            // dt <= nsub CFL dx / c_hat: nsub substeps of dt / nsub respect the radiation CFL
    rc = do_hydro_step(c, 1.0, &c->ddt->dtdx);
    for (int s = 0; s < nsub && rc == QK_OK; ++s) {
        rc = do_rad_transport(c, 1.0, &c->ddt->dtsdx);
        if (rc == QK_OK) rc = do_exchange(c, 1.0, &c->ddt->dts);
    }
    c->last_nsub = nsub;
    return rc;
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

// ---- replayable step: one qk_hydro_step_cfl / qk_rhd_step_cfl recorded as a CUDA graph ------------------------
// The launch sequence of a step depends on the host-side state only (parameters, boundary types, which caches are
// valid), never on device data -- the timestep stays on the device -- so a step recorded once in the steady state
// (reconstruction variables and CFL speed left by the previous step) is the step, whatever the data.
int qk_graph_free(qk_ctx *c)
{
    if (!c) return QK_EINVAL;
    if (c->graph.exec) { cudaGraphExecDestroy(c->graph.exec); c->graph.exec = nullptr; }
    return QK_OK;
}

int qk_graph_capture(qk_ctx *c, int kind, int nsub)
{
    if (!c || (kind != QK_GRAPH_HYDRO && kind != QK_GRAPH_RHD)) return QK_EINVAL;
    if (kind == QK_GRAPH_RHD && (nsub < 1 || nsub > c->pc.nsub_max || !(c->pc.c_hat > 0.0) || !(c->pc.c > 0.0))) return QK_EINVAL;
    if (c->ext_faces || c->profiling || c->halo_failed) return QK_EINVAL;
    int rc = ensure_storage(c);
    if (rc) return rc;
    qk_graph_free(c);
    // record the steady-state sequence: as if the previous step had left its caches (a launch on a context whose
    // caches are not valid takes one ordinary step instead, qk_graph_launch)
    const bool w = c->w_valid, sv = c->s_valid, sm = c->smax_valid;
    const long long launches0 = c->launches;
    const int nsub0 = c->last_nsub;
    c->w_valid = c->s_valid = c->smax_valid = true;
    if (cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
        cudaGetLastError();                      // e.g. the legacy default stream cannot be captured
        c->w_valid = w; c->s_valid = sv; c->smax_valid = sm;
        return QK_EINVAL;
    }
    rc = kind == QK_GRAPH_HYDRO ? qk_hydro_step_cfl(c) : qk_rhd_step_cfl(c, nsub);
    cudaGraph_t g = nullptr;
    const cudaError_t e = cudaStreamEndCapture(c->stream, &g);
    const int per_step = (int)(c->launches - launches0);
    c->w_valid = w; c->s_valid = sv; c->smax_valid = sm; c->launches = launches0; c->last_nsub = nsub0;
    if (rc != QK_OK || e != cudaSuccess || !g) {
        if (g) cudaGraphDestroy(g);
        cudaGetLastError();
        return rc != QK_OK ? rc : QK_ECUDA;
    }
    cudaGraphExec_t exec = nullptr;
    const cudaError_t ei = cudaGraphInstantiate(&exec, g, 0);
    cudaGraphDestroy(g);
    if (ei != cudaSuccess) { cudaGetLastError(); return QK_ECUDA; }
    c->graph.exec = exec; c->graph.kind = kind; c->graph.nsub = kind == QK_GRAPH_RHD ? nsub : 0; c->graph.launches = per_step;
    c->graph.pc = c->pc; c->graph.fb = c->fb; c->graph.has_fixed = c->has_fixed; c->graph.has_source = c->has_source;
    c->graph.chi_path = c->chi_path; c->graph.stream = c->stream; c->graph.base = c->base;
    return QK_OK;
}

int qk_graph_launch(qk_ctx *c, int nsteps)
{
    if (!c || !c->graph.exec || nsteps < 0) return QK_EINVAL;
    const qk_ctx::StepGraph &G = c->graph;
    // recorded for other parameters, boundaries, storage or stream than the context has now: record again
    if (memcmp(&G.pc, &c->pc, sizeof(PhysConsts)) != 0 || memcmp(&G.fb, &c->fb, sizeof(FaceBc)) != 0 ||
        G.has_fixed != c->has_fixed || G.has_source != c->has_source || G.chi_path != c->chi_path ||
        G.stream != c->stream || G.base != c->base || c->ext_faces || c->profiling || c->halo_failed) return QK_EINVAL;
    for (int n = 0; n < nsteps; ++n) {
        const bool steady = c->smax_valid && (c->has_fixed || (c->w_valid && (G.kind == QK_GRAPH_HYDRO || c->s_valid)));
        if (!steady) {                           // fresh state: the ordinary step builds the caches the graph starts from
            const int rc = G.kind == QK_GRAPH_HYDRO ? qk_hydro_step_cfl(c) : qk_rhd_step_cfl(c, G.nsub);
            if (rc) return rc;
            continue;
        }
        if (cudaGraphLaunch(G.exec, c->stream) != cudaSuccess) { cudaGetLastError(); return QK_ECUDA; }
        c->launches += G.launches;
        c->last_nsub = G.nsub;
    }
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
    const bool cfl_bad = c->smax_valid && sc.cfl_bad != 0;     // set by the last qk_cfl_dt / hydro step / exchange
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

int qk_set_flatten_path(qk_ctx *c, int path)
{
    if (!c || path < 0 || path > 2) return QK_EINVAL;
    c->chi_path = path;
    return QK_OK;
}

int qk_kernel_class_count(void) { return K_NCLASS; }

const char *qk_kernel_class_name(int cls)
{
    static const char *names[K_NCLASS] = {"fill_boundary", "cfl", "flatten", "hydro_sweep_x", "hydro_sweep_y", "hydro_sweep_z", "rad_sweep_x",
                                          "rad_sweep_y", "rad_sweep_z",
                                          "exchange", "opacity", "prim", "halo"};
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

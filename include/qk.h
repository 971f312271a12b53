/* qk.h -- C ABI of the B200-native per-timestep uniform-grid cell update of the QUOKKA
 * method (Wibking & Krumholz, arXiv:2110.01792).  Citations are /root/reference/PAPER.md
 * line numbers ("PAPER.md:<line>") and DESIGN.md readings (H*, R*, X*).
 *
 * One context = one uniform box of nx*ny*nz cells with QK_NG ghost zones per side on one
 * GPU, fp64, structure-of-arrays.  Every field is a dense array of
 * (nz+2*QK_NG)*(ny+2*QK_NG)*(nx+2*QK_NG) doubles, x fastest; interior cell (i,j,k),
 * 0-based, sits at ((k+QK_NG)*(ny+2*QK_NG) + (j+QK_NG))*(nx+2*QK_NG) + (i+QK_NG).
 *
 * All step functions run hand-written sm_100a CUDA kernels; there is no CPU fallback.
 * They are asynchronous on the context's stream and return QK_OK once enqueued (or the
 * CUDA launch error).  State errors found on the device (non-positive density, pressure
 * or radiation energy; Newton failure) are counted there and surfaced by qk_last_info,
 * which synchronises.  No function calls exit(); no global state; contexts are independent.
 *
 * Pointer arguments named `interior`/`with_ghosts` may be HOST or DEVICE pointers (the
 * library asks the CUDA runtime which); set/get copy and never alias the caller's array.
 */
#ifndef QK_H
#define QK_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define QK_NG 4   /* ghost zones per side: PPM needs 3, multidimensional flattening 4 (H6) */

typedef struct qk_ctx qk_ctx;   /* opaque; owns layout, stage buffers, device counters */

enum { QK_OK = 0, QK_EINVAL = 1, QK_ENOMEM = 2, QK_ECUDA = 3,
       QK_ENEWTON = 4,   /* >=1 cell hit the Newton iteration cap              */
       QK_ESTATE = 5 };  /* rho<=0, P<=0, E_g<=0 or E_r<=0 met (PAPER.md:438 needs E_r>0)      */

enum { QK_BC_PERIODIC = 0,
       QK_BC_OUTFLOW = 1,    /* PAPER.md:464; zero-gradient copy of the nearest interior cell (H15) */
       QK_BC_REFLECTING = 2, /* PAPER.md:408, 438, 464; solid wall: mirror image, the wall-normal component of
                                rho v and F_r negated (B1) */
       QK_BC_FIXED = 3 };    /* Dirichlet / inflow: the ghost cells beyond the
                                face keep the values the caller stored with qk_set_raw (B2) */

/* field ids: conserved hydro U=(rho, rho v, E), radiation moments
 * (E_r, F_r) (eq 11-12), Planck- and Rosseland-type opacities per cell
 * (kappa_E~kappa_P, kappa_F~kappa_R), static during a step. */
enum { QK_RHO = 0, QK_MX, QK_MY, QK_MZ, QK_E, QK_ER, QK_FX, QK_FY, QK_FZ, QK_KAPPA_P, QK_KAPPA_R,
       QK_SRC,      /* radiation energy source rate per cell (e.g. stellar sources): the S of eq 27 / 38 is dt * src
                       (reading X13); zero unless set; read by the exchange step only */
       QK_NFIELDS };

enum { QK_FLAG_TAU_CORR = 1,        /* guarded optical-depth correction of the E_r HLL flux in the form
                                       of reading R6.  OFF by default: the paper prints no formula and this form misses
                                       the one number it prints for tau_cell >> 1 (R6)        */
       QK_FLAG_STATIC_MATTER = 2,   /* exchange skips eq 41-43: gas held at rest (X11)            */
       QK_FLAG_NEWTON_LITERAL = 4,  /* literal stop rule of PAPER.md:237 instead of converge-then-polish (X5)   */
       /* scheme variants: */
       QK_FLAG_PLM = 8,             /* piecewise-linear reconstruction, monotonized-central limiter, for hydro
                                       and radiation instead of PPM                              */
       QK_FLAG_EDDINGTON = 16,      /* Eddington approximation chi = 1/3, P_r = E_r/3,
                                       instead of the Levermore closure                                         */
       QK_FLAG_MINERBO = 32 };      /* Minerbo (1978) closure in the APPROXIMATE polynomial form customary in the
                                       literature, chi = 1/3 + (2/15) f^2 (3 - f + 3 f^2) (within 0.011 of the
                                       maximum-entropy definition; PAPER.md:196 names the closure, prints no formula;
                                       V3); not together with QK_FLAG_EDDINGTON                                 */

enum { QK_FILL_HYDRO = 1, QK_FILL_RAD = 2, QK_FILL_OPACITY = 4, QK_FILL_ALL = 7 };

/* z-slab domain decomposition (one box per GPU; the paper's pattern: one ghost exchange per
 * RK stage).  Faces named here border another rank's slab. */
enum { QK_FACE_ZLO = 1, QK_FACE_ZHI = 2 };
typedef int (*qk_halo_fn)(void *user, int nfields);   /* 0 = ok; anything else aborts the step with QK_EINVAL */

/* Counters of the most recent step call (qk_hydro_step / qk_rad_step / qk_rhd_step / qk_exchange
 * / qk_rad_transport), summed over the substeps of a qk_rhd_step. */
typedef struct qk_info {
    int       nsub;               /* radiation substeps taken by the last qk_rhd_step */
    int       newton_max_iters;   /* largest Newton iteration count in any cell                      */
    long long newton_fail_cells;  /* cells that reached newton_maxit without converging              */
    long long newton_total_iters; /* sum of iteration counts over cells                               */
    long long bad_state_cells;    /* cells flagged QK_ESTATE                                           */
    long long fallback_states;    /* radiation face states reverted to first order     */
    long long guard_faces;        /* faces where the tau correction was disabled       */
    int       status;             /* QK_OK, QK_ENEWTON or QK_ESTATE                                   */
} qk_info;

/* Create a context for an nx*ny*nz box (each >= 1), cell size dx, adiabatic index gamma,
 * reduced and physical speeds of light c_hat, c (eq 13-17; pass 0,0 for pure
 * hydro) and boundary QK_BC_*.  Selects the current CUDA device.  Device memory for the
 * state is allocated here with cudaMalloc unless `qk_bind_storage` supplies it before
 * first use (allocation is deferred to first use).  Defaults: a_rad = 1, k_B/(mu m_H) = 1,
 * CFL 0.3, Newton tolerance 1e-10, 400 iterations, N_sub,max 10,
 * flags = 0.  Returns QK_EINVAL / QK_ENOMEM / QK_ECUDA on failure. */
int qk_init(int nx, int ny, int nz, double dx, double gamma, double c_hat, double c, int boundary,
            qk_ctx **out);

/* Destroy a context; frees device memory the library allocated (never bound storage). */
int qk_free(qk_ctx *ctx);

/* Bytes of device memory one context needs (12 state fields, 5 RK stage fields, the flattening
 * coefficient, 5 flux-difference accumulators, two sets of primitives and of radiation reconstruction
 * variables and counters: 44 fields), for
 * callers that own the allocation (torch.empty). */
size_t qk_state_bytes(int nx, int ny, int nz);

/* Use caller-owned DEVICE memory (>= qk_state_bytes, 256-byte aligned) instead of
 * cudaMalloc.  Must precede the first set/get/step call.  The caller keeps ownership. */
int qk_bind_storage(qk_ctx *ctx, void *dev_ptr, size_t bytes);

/* cudaStream_t (as void*) all later work of this context is enqueued on; NULL = default. */
int qk_set_stream(qk_ctx *ctx, void *cuda_stream);

/* radiation constant a_r and k_B/(mu m_H) of the ideal-gas temperature
 * T = (gamma-1) E_g / (rho k_B/(mu m_H)) (X2). */
int qk_set_constants(qk_ctx *ctx, double a_rad, double kB_over_mu_mH);

/* Boundary type per face, in the order x-lo, x-hi, y-lo, y-hi, z-lo, z-hi (qk_init sets all six alike).  Periodic
 * must be given on both faces of an axis (QK_EINVAL otherwise).  A ghost cell takes, axis by axis, the rule of the
 * face its index lies beyond; a cell beyond any QK_BC_FIXED face is never written by the fill: store its values
 * (all state fields, the whole ghost slab including edges and corners) with qk_set_raw before stepping. */
int qk_set_face_boundaries(qk_ctx *ctx, const int *bc6);

/* Density power-law opacities kappa_P,R = kappa0_P,R (rho/rho0)^exponent, integer exponent in [-4, 4] (the laws of
 * the paper's tests: rho kappa ~ rho^2; kappa ~ 1/rho; X14).  When rho0 > 0 the two
 * opacity fields of the interior cells are recomputed from the current density at the start of every radiation
 * subcycle; rho0 = 0 (default) leaves the fields as the caller set them. */
int qk_set_opacity_law(qk_ctx *ctx, double kappaP0, double kappaR0, double rho0, int exponent);

/* The same law times (T/T0)^(texp2/2), T the gas temperature and texp2 an integer in [-16, 16]: half-integer powers
 * such as Kramers' kappa ~ rho T^-3.5 (exponent 1, texp2 -7), evaluated by repeated multiplication and one square
 * root.  With texp2 != 0 the exchange treats kappa_P implicitly -- it follows the temperature of the Newton iterate
 * and enters the Jacobian through the d kappa_P/dT term of eq 33 -- and takes kappa_F ~ kappa_R at the
 * updated temperature; the opacity fields are refreshed from (rho, T) before every transport step. */
int qk_set_opacity_law_T(qk_ctx *ctx, double kappaP0, double kappaR0, double rho0, int exponent, double T0, int texp2);

/* Equation of state of the gas in the EXCHANGE step: QK_EOS_IDEAL (default; T = (gamma-1) E_g / (rho k_B/(mu m_H)))
 * or QK_EOS_ALPHA_T3, E_g = alpha T^4 / 4 with volumetric heat capacity C_v = alpha T^3 (eq 55, PAPER.md:424-427;
 * the Marshak, Su-Olson and energy-exchange tests, where the matter is static).  The hydro step always uses the
 * ideal gas. */
enum { QK_EOS_IDEAL = 0, QK_EOS_ALPHA_T3 = 1 };
int qk_set_eos(qk_ctx *ctx, int eos, double alpha);

/* CFL number C0/D of eq 21, Newton tolerance and iteration cap,
 * N_sub,max and QK_FLAG_* bits. */
int qk_set_params(qk_ctx *ctx, double cfl, double newton_tol, int newton_maxit, int nsub_max,
                  unsigned flags);

/* Copy one field's interior, nz*ny*nx doubles x fastest (host or device), into / out of the
 * state.  qk_get_state synchronises the stream before returning. */
int qk_set_state(qk_ctx *ctx, int field, const double *interior);
int qk_get_state(qk_ctx *ctx, int field, double *interior);

/* The same for n fields at once WITHOUT synchronising: one copy per field on the context's own copy stream, ordered
 * against the compute stream by events (an upload waits for the compute work enqueued so far and the next step waits
 * for the upload; a download waits for the steps enqueued so far).  interiors[m] belongs to fields[m]; host arrays
 * should be pinned (pageable memory still works but the copies then serialise) and must stay untouched until
 * qk_wait_copies returns.  With two contexts the upload of one box, the step of the other and the download of the
 * previous result overlap. */
int qk_set_state_all(qk_ctx *ctx, int n, const int *fields, const double *const *interiors);
int qk_get_state_all(qk_ctx *ctx, int n, const int *fields, double *const *interiors);
int qk_wait_copies(qk_ctx *ctx);

/* Same with the ghost zones: (nz+8)(ny+8)(nx+8) doubles (boundary-fill parity checks, Dirichlet values).  The
 * step functions fill the ghost zones of their internal reconstruction variables, not necessarily those of the
 * state fields: call qk_fill_boundary first to see the boundary images of the current state. */
int qk_set_raw(qk_ctx *ctx, int field, const double *with_ghosts);
int qk_get_raw(qk_ctx *ctx, int field, double *with_ghosts);

/* Fill the ghost shell (faces, edges, corners) of the field groups in `which` (QK_FILL_*):
 * every ghost cell <- the interior cell its three indices map to, periodic wrap or
 * nearest-interior copy ("B.C. fill"). */
int qk_fill_boundary(qk_ctx *ctx, int which);

/* Declare the z faces in `faces` (QK_FACE_* bits) as inter-rank faces.  Before every ghost fill the library then
 * calls fn(user, nfields) on the calling thread; inside it the caller moves the halos of the nfields fields about
 * to be filled: qk_halo_pack(face, buf) copies the QK_NG interior planes next to `face` of each of them into the
 * DEVICE buffer buf (nfields * qk_halo_doubles() doubles, field-major, planes ascending in z, ny*nx interior cells
 * per plane), the caller sends it to the neighbour (NCCL send/recv, peer copy, ...), and qk_halo_unpack(face, buf)
 * writes a received buffer into the QK_NG ghost planes beyond `face`.  All on the context's stream.  After fn
 * returns the library fills the remaining ghost cells (x, y images and the physical z faces).  The result equals
 * the single-box update bit for bit.  faces = 0 or fn = NULL switches the decomposition off.  Needs nz >= QK_NG.
 * qk_halo_pack / qk_halo_unpack return QK_EINVAL outside the callback.  qk_cfl_dt stays local: the caller takes
 * the minimum over ranks. */
int qk_set_halo_exchange(qk_ctx *ctx, unsigned faces, qk_halo_fn fn, void *user);
size_t qk_halo_doubles(const qk_ctx *ctx);          /* QK_NG * ny * nx: doubles per field per face */
int qk_halo_pack(qk_ctx *ctx, int face, double *dev_buf);
int qk_halo_unpack(qk_ctx *ctx, int face, const double *dev_buf);

/* The same decomposition WITHOUT the host on the stage path: every rank maps its neighbours' storage (CUDA IPC between
 * processes, plain pointers inside one process) and, before a ghost fill, a kernel on a side stream writes its
 * QK_NG boundary planes straight into the neighbour's ghost planes (NVLink / NVSwitch peer stores) and raises an arrival
 * counter in the neighbour's memory; the consuming stream waits on its own counter with a stream memory operation.
 * Nothing spins and no host thread waits.  Each RK stage is ordered so that everything that reads no z ghost plane (the
 * x / y images of the interior planes, flattening and x / y sweeps of the planes >= 3 cells from the faces; for
 * radiation all x / y sweeps) runs while the planes travel; only the remaining boundary work and the z sweep wait
 * (the paper attributes its multi-GPU loss to ghost fills that are not overlapped).
 *   qk_halo_export    : describe this context's storage (after qk_bind_storage, if used).  Synchronises.
 *   qk_set_halo_peers : attach the neighbour below (lo) and above (hi) in z; NULL = physical boundary on that face.
 *                       Every rank exports, the handles are exchanged (e.g. torch.distributed.all_gather_object), every
 *                       rank attaches, and only then does any rank step (the arrival counters restart at attach).  All
 *                       ranks must then make the same sequence of step / fill calls.  Needs nz >= QK_NG, equal nx, ny;
 *                       nz may differ between ranks.  (NULL, NULL) detaches.  qk_cfl_dt stays local: the caller takes
 *                       the minimum over ranks.  The result equals the single-box update bit for bit.  QK_EINVAL when
 *                       the driver has no stream memory operations (use qk_set_halo_exchange then). */
typedef struct qk_halo_handle {
    unsigned char ipc[64];        /* cudaIpcMemHandle_t of the allocation that holds the storage (has_ipc != 0)    */
    unsigned long long base;      /* device address of the storage in the exporting process                        */
    unsigned long long offset;    /* of the storage inside that allocation                                         */
    long long pid;                /* exporting process: handles of the same process are attached by address        */
    int device, nx, ny, nz, has_ipc;
} qk_halo_handle;
int qk_halo_export(qk_ctx *ctx, qk_halo_handle *out);
int qk_set_halo_peers(qk_ctx *ctx, const qk_halo_handle *lo, const qk_halo_handle *hi);

/* eq 21: dt = CFL dx / max_cells(|v| + c_s), |v| the vector magnitude,
 * further limited to nsub_max CFL dx / c_hat when c_hat > 0.  Synchronises.
 * Returns NaN if a cell has rho <= 0 or P <= 0 (then qk_last_info().status = QK_ESTATE). */
double qk_cfl_dt(qk_ctx *ctx);

/* One SSP-RK2 method-of-lines hydro step: per stage ghost fill,
 * primitives, multidimensional flattening, PPM face states, HLLC fluxes, unsplit update. */
int qk_hydro_step(qk_ctx *ctx, double dt);

/* The same step with the timestep of eq 21 (qk_cfl_dt's formula and CFL number) evaluated ON THE DEVICE from the
 * signal speed the previous step left there: nothing is read back, the launch queue never drains.  qk_last_dt
 * returns the dt that was used (synchronises).  If the state is bad (rho <= 0 or P <= 0 somewhere) dt is NaN, the
 * state becomes NaN and qk_last_info().status is QK_ESTATE.  QK_EINVAL on a context with inter-rank faces (a slab's
 * own signal speed is not the global one: take qk_cfl_dt, reduce over ranks, call qk_hydro_step). */
int qk_hydro_step_cfl(qk_ctx *ctx);
int qk_last_dt(qk_ctx *ctx, double *dt);

/* The coupled cycle of qk_rhd_step with the device-resident timestep: dt = min(CFL dx / max(|v| + c_s),
 * nsub CFL dx / c_hat), so that the nsub radiation substeps of dt / nsub the caller asks for respect the radiation
 * CFL condition; 1 <= nsub <= nsub_max.  Same trajectory as qk_cfl_dt + qk_rhd_step whenever
 * that pair would take nsub substeps of the same dt. */
int qk_rhd_step_cfl(qk_ctx *ctx, int nsub);

/* Replayable step: ONE qk_hydro_step_cfl (kind QK_GRAPH_HYDRO) or ONE qk_rhd_step_cfl(nsub) (kind QK_GRAPH_RHD)
 * recorded as a CUDA graph and replayed with one launch per step.  The launch sequence of a step is fixed by the
 * host-side parameters alone (the timestep of eq 21 stays on the device), so the recorded step is
 * the same kernels with the same arguments as the ordinary call: results are bit-identical.  For boxes below ~128^3 the
 * step is bound by launch overhead and the replay removes it.
 * qk_graph_capture records the steady-state sequence on the context's stream, which must not be the legacy default
 * stream (QK_EINVAL: it cannot be captured); nothing is executed and the state is not touched.  It replaces an
 * earlier recording.  QK_EINVAL also for a context with inter-rank faces (see qk_hydro_step_cfl) or with kernel-class
 * timing on.  Allocation happens here (graph instantiation), never in qk_graph_launch.
 * qk_graph_launch enqueues `nsteps` steps.  A step whose starting state has no cached reconstruction variables
 * (the first step after qk_set_state / qk_set_raw) is taken by the ordinary call instead, which builds them.
 * QK_EINVAL if nothing was recorded or if parameters, boundary types, opacity law, equation of state, source field,
 * flattening path, storage or stream have changed since the recording: record again.  Counters (qk_last_info) are
 * those of the last step; qk_last_dt returns its dt.
 * qk_graph_free drops the recording (qk_free does too). */
#define QK_GRAPH_HYDRO 0
#define QK_GRAPH_RHD 1
int qk_graph_capture(qk_ctx *ctx, int kind, int nsub);
int qk_graph_launch(qk_ctx *ctx, int nsteps);
int qk_graph_free(qk_ctx *ctx);

/* SSP-RK2 explicit transport of (E_r, F_r) over dt, no exchange. */
int qk_rad_transport(qk_ctx *ctx, double dt);

/* Per-cell implicit matter-radiation exchange over dt (eq 26-43). */
int qk_exchange(qk_ctx *ctx, double dt);

/* ONE radiation subcycle: qk_rad_transport(dt) then qk_exchange(dt). */
int qk_rad_step(qk_ctx *ctx, double dt);

/* Operator-split cycle: hydro step, then N_sub = max(1, ceil(dt c_hat /
 * (CFL dx))) radiation subcycles of dt/N_sub.  QK_EINVAL if N_sub > nsub_max. */
int qk_rhd_step(qk_ctx *ctx, double dt);

/* Number of radiation substeps qk_rhd_step(dt) would take. */
int qk_nsub_for(const qk_ctx *ctx, double dt);

/* Synchronise and report the counters of the last step call. */
int qk_last_info(qk_ctx *ctx, qk_info *out);

/* Number of kernel launches this context has enqueued so far (bench.py's gpu_launches). */
long long qk_launch_count(const qk_ctx *ctx);

/* Per-kernel-class device timing for the roofline report.  While
 * profiling is on, every group of launches of one kernel class is bracketed by CUDA events on
 * the context's stream.  qk_kernel_times synchronises, adds the elapsed ms and the number of
 * bracketed groups per class into ms[]/count[] (arrays of qk_kernel_class_count() entries) and
 * clears the record. */
int qk_set_profiling(qk_ctx *ctx, int on);

/* Which implementation of the flattening coefficient (H6) a hydro stage launches:
 * 0 = by box size (default), 1 = two pointwise passes through three chi~ arrays (faster while those stay in
 * L2, boxes up to ~160^3), 2 = one z-marching pass without chi~ arrays (half the HBM bytes; faster beyond).
 * Both give the same bits; the switch exists so that tests and measurements can run either on any box.
 * QK_EINVAL for another value. */
int qk_set_flatten_path(qk_ctx *ctx, int path);
int qk_kernel_class_count(void);
const char *qk_kernel_class_name(int cls);
int qk_kernel_times(qk_ctx *ctx, double *ms, long long *count);

/* fp64 pipe throughput probe (roofline denominator of the ALU-bound stage kernels, DESIGN.md
 * section 6): kind 0 = dependent DMUL+DADD chains (the -fmad=false mix the library computes in),
 * kind 1 = DFMA chains.  Writes fp64 instructions x 32 lanes per second.  Synchronises. */
int qk_fp64_probe(int kind, int iters, void *cuda_stream, double *lane_ops_per_s);

/* Self-test of the library's branch-free fp64 division and square root (used inside the Riemann
 * solvers of the sweep kernels): n seeded random operand pairs with exponents
 * spread over `exponent_span` binades centred on 1 (2046 = every normal double; zeros, subnormals,
 * infinities and NaNs are mixed in).  out4 = {divisions accepted by the range test, of those not
 * bit-equal to IEEE x/y, square roots accepted, of those not bit-equal to IEEE sqrt}.  Synchronises. */
int qk_selftest_divsqrt(long long n, unsigned long long seed, int exponent_span, void *cuda_stream,
                        long long *out4);

/* ---- Allocation-free entry point -------------------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it): the hydro timestep of eq 21, dt = cfl * dx / max_cells(|v| + c_s), of a DENSE state, with
 * no context and no allocation of any kind.  rho, mx, my, mz, E: DEVICE pointers to ncells contiguous doubles each
 * (conserved variables, any cell order, no ghost cells; read only).  dt_out: DEVICE pointer to one double, written
 * by the last kernel (NaN if a cell has rho <= 0 or P <= 0).  Asynchronous on cuda_stream (a cudaStream_t; NULL =
 * the default stream); nothing is read back, nothing synchronises.  The value equals qk_cfl_dt's bit for bit on the
 * same cells (with c_hat = 0: there is no radiation limit here).
 * Scratch: one partial maximum per 1024 cells and a bad-cell counter live in a file-scope device array of
 * QK_NOALLOC_SCRATCH_BYTES that every GPU loading the library holds until exit; hence the limit
 * ncells <= QK_NOALLOC_MAX_CELLS (256^3), beyond which the call returns QK_ENOMEM and launches nothing.
 * QK_EINVAL for a null pointer, ncells < 1, gamma <= 1, cfl <= 0 or dx <= 0; QK_ECUDA if a CUDA call fails.
 * The array is shared by every call in the process and keeps the last call's contents (the call clears the counter
 * it needs at zero itself): calls that may overlap on the GPU -- different streams, several host threads -- race on
 * it and must be serialised by the caller.
 * qk_noalloc_setup resolves the array's device address for the CURRENT device (cudaGetSymbolAddress, once per
 * device); qk_cfl_dt_noalloc does the same on first use, so calling it is only needed before a region in which
 * even that query is unwelcome (stream capture).  qk_noalloc_max_cells returns QK_NOALLOC_MAX_CELLS. */
#define QK_NOALLOC_MAX_CELLS 16777216LL
#define QK_NOALLOC_SCRATCH_BYTES 131328
int qk_noalloc_setup(void);
long long qk_noalloc_max_cells(void);
int qk_cfl_dt_noalloc(const double *rho, const double *mx, const double *my, const double *mz, const double *E,
                      long long ncells, double gamma, double cfl, double dx, void *cuda_stream, double *dt_out);

const char *qk_version(void);

#ifdef __cplusplus
}
#endif
#endif /* QK_H */

/* kharm.h -- C ABI of libkharm.so: the B200 (sm_100a) hot path of the KHARMA/HARM method.
 *
 * One explicit second-order (predictor-corrector) ideal-GRMHD update of a uniform logically
 * Cartesian 3-D mesh block in a stationary metric, fp64, entirely in hand-written CUDA kernels.
 * There is NO CPU fallback: every call that computes needs a CUDA device and fails with KH_ECUDA
 * otherwise.
 *
 * Citations: "P:n" = PAPER.md line n.  The paper gives the scheme by citation (P:243 HARM, the
 * modified 3-velocity, the 1D_W inversion, Flux-CT; P:253 MC / WENO5; P:255 predictor-corrector;
 * P:111 FMKS; P:257-261 floors; P:317 the sub-step's task list) and prints eq. 1.1; the
 * exact formulas adopted are the readings S1..S23 listed in DESIGN.md.
 *
 * Conventions
 *   - primitives, 8 per zone: rho, u, ut^1, ut^2, ut^3, B^1, B^2, B^3  (ut = the velocity of P:243)
 *   - arrays are fp64, SoA [var][k][j][i], x1 (i) fastest, C order, densely packed
 *       with_ghosts = 0 : [8][n3][n2][n1]            interior only
 *       with_ghosts = 1 : [8][n3+6][n2+6][n1+6]      KH_NG = 3 ghost layers per side in all directions
 *   - `mem` says where a caller buffer lives: KH_MEM_DEVICE (a device pointer valid on the grid's
 *     device; copies are enqueued on the grid's stream) or KH_MEM_HOST (a host pointer; the call
 *     copies through the stream and returns after the copy completed)
 *   - ownership: the library owns the grid and all internal buffers; callers own every buffer they pass
 *   - errors: every call returns KH_OK (0) or a negative code; no exceptions or aborts cross the ABI;
 *     out-parameters are untouched on error.  U->P failures are DATA (pflag), not errors.
 *   - threading: calls on one grid must be serialised by the caller; all work is enqueued on the
 *     grid's stream: the one given at creation, or, for NULL, a blocking stream the grid creates for
 *     itself (the legacy default stream cannot be captured into a CUDA graph).  That own stream orders
 *     against the legacy default stream only; callers on other streams order against the grid with
 *     kh_get_stream / kh_sync.  KH_MEM_DEVICE transfers and kh_step(..., NULL) return without waiting.
 *   - device: a grid lives on the CUDA device that was current at kh_grid_create; every call makes that
 *     device current for the calling thread.
 */
#ifndef KHARM_H
#define KHARM_H
#ifdef __cplusplus
extern "C" {
#endif

#define KH_NG 3
#define KH_NPRIM 8

enum { KH_OK = 0, KH_EINVAL = -1, KH_ENOMEM = -2, KH_ECUDA = -3, KH_ENAN = -4,
       KH_ESIZE = -5 /* kh_divB_noalloc: more corners than its static scratch covers (KH_NOALLOC_MAX_CORNERS) */ };
enum { KH_MINKOWSKI = 0, KH_KS = 1, KH_FMKS = 2 };                            /* coords          */
enum { KH_BC_PERIODIC = 0, KH_BC_OUTFLOW = 1, KH_BC_POLAR = 2, KH_BC_FIXED = 3,
       KH_BC_BLOCK = 4 /* ghost layers owned by a neighbouring block: kh_link_blocks, kh_step_blocks */ };
enum { KH_RECON_MC = 0, KH_RECON_WENO5 = 1 };
enum { KH_INV_1DW = 0, KH_INV_KASTAUN = 1 };
enum { KH_FRAME_FLUID = 0, KH_FRAME_DRIFT = 1, KH_FRAME_NORMAL = 2 };
enum { KH_B_FLUX_CT = 0, KH_B_FACE_CT = 1 };
enum { KH_EMF_ARITHMETIC = 0, KH_EMF_UPWIND = 1, KH_EMF_CENTRED = 2 };
enum { KH_MEM_DEVICE = 0, KH_MEM_HOST = 1 };
enum { KH_LOC_CENT = 0, KH_LOC_FACE1 = 1, KH_LOC_FACE2 = 2, KH_LOC_FACE3 = 3 };

typedef struct {
  int coords;                 /* KH_MINKOWSKI (Cartesian) | KH_KS (native = r,theta,phi) | KH_FMKS */
  double a;                   /* black-hole spin (KS / FMKS)                                               */
  double hslope, poly_xt, poly_alpha, mks_smooth;   /* FMKS map parameters (poly_alpha: even integer value) */
  int n1, n2, n3;             /* interior zones; n3 == 1 runs a 2-D problem as a one-zone-thick block      */
  double xmin[3], xmax[3];    /* native-coordinate bounds of the interior                                  */
  int bc[6];                  /* x1lo x1hi x2lo x2hi x3lo x3hi; periodic must be set on both sides;
                                 KH_BC_POLAR only in x2 (needs n2 >= 3); KH_BC_BLOCK needs N_d >= 3          */
  double gamma, cfl;          /* adiabatic index; Courant factor                                           */
  int recon;                  /* KH_RECON_MC | KH_RECON_WENO5                                              */
  double rho_min, u_min, r_char, bsq_over_rho_max, bsq_over_u_max, u_over_rho_max, gamma_max; /* floors */
  double dt_growth_max;       /* dt_next <= dt_growth_max * dt                                              */
  int inverter;               /* KH_INV_1DW (the 1D_W Newton iteration) | KH_INV_KASTAUN (the
                                 bracketed root find of Kastaun et al.; same pflag codes, no guess needed)   */
  int fofc;                   /* 1: first-order flux correction: a speculative update finds the zones
                                 that would fail the inversion or hit a floor; their faces get donor-cell LLF fluxes */
  int floor_frame;            /* frame the floor material is injected in: KH_FRAME_FLUID (velocity
                                 untouched) | KH_FRAME_DRIFT (E x B drift velocity kept, momentum along B conserved) |
                                 KH_FRAME_NORMAL (added as gas at rest for the normal observer, then re-inverted)   */
  int transport;              /* magnetic field transport: KH_B_FLUX_CT (zone-centred field, Toth's Flux-CT) |
                                 KH_B_FACE_CT (face-centred field advanced by the circulation of the edge EMFs;
                                 needs kh_set_face_B)                                                          */
  int emf;                    /* edge EMFs of either transport ("a number of schemes ... with and without upwinding"):
                                 KH_EMF_ARITHMETIC (four-point average of the face fluxes) | KH_EMF_UPWIND (Gardiner & Stone,
                                 contact-upwinded) | KH_EMF_CENTRED (Gardiner & Stone without upwinding: half the sum of the
                                 four face values minus a quarter of the sum of the four zone-centred values)    */
} kh_params;

typedef struct kh_grid kh_grid;   /* opaque */

/* Create a grid on the current CUDA device and run the one-time geometry precompute (kernel K1:
 * gcov, gcon, sqrt(-g), lapse at zone centres and the three face centres, connection coefficients
 * and floor profiles at centres; the "caches of expensive-to-calculate quantities" of P:285).
 * cuda_stream: a cudaStream_t (as void*), or NULL: the grid then creates its own blocking stream.
 * Errors: KH_EINVAL for parameters out of range, also for a block of 2^31 or more zones with ghosts (zone numbers are held
 * in 32 bits; one state array of such a block would not fit a device); KH_ENOMEM; KH_ECUDA. */
int kh_grid_create(const kh_params* params, void* cuda_stream, kh_grid** out);
int kh_grid_destroy(kh_grid* g);
/* The stream every call on this grid enqueues on (a cudaStream_t as void*), and a wait for all of it. */
int kh_get_stream(kh_grid* g, void** cuda_stream);
int kh_sync(kh_grid* g);

/* Load primitives and fill the ghost zones (periodic / outflow / polar as configured; KH_BC_FIXED
 * ghosts keep what a with_ghosts = 1 array supplies).  Kernel K7.
 * A grid with a KH_BC_FIXED side needs one with_ghosts = 1 load before anything else: until then
 * kh_set_prims(with_ghosts = 0) and kh_step return KH_EINVAL (the fixed layers would be vacuum).
 * On a face-centred CT grid whose face field has been set (kh_set_face_B), the face field remains the
 * magnetic state: the B components of p are replaced by the face means. */
int kh_set_prims(kh_grid* g, const double* p, int with_ghosts, int mem);
int kh_get_prims(kh_grid* g, double* p, int with_ghosts, int mem);

/* Conserved variables U(P) = sqrt(-g)(rho u^t, T^t_t + rho u^t, T^t_i, B^i) at zone centres,
 * interior [8][n3][n2][n1] (T from eq. 1.1). */
int kh_get_cons(kh_grid* g, double* u, int mem);

/* Flags of the LAST sub-step, interior [n3][n2][n1], as int32.  pflag: 0 ok, 1 bad input,
 * 2 no convergence, 3 v^2 out of range, 4 rho <= 0, 5 u < 0, 6 both, 7 non-finite (1D_W inversion,
 * P:243).  fflag: bits 1 rho geometric floor, 2 rho b^2 floor, 4 u geometric floor, 8 u b^2 floor,
 * 16 u/rho ceiling, 32 Lorentz-factor ceiling.  Either pointer may be NULL. */
int kh_get_flags(kh_grid* g, int* pflag, int* fflag, int mem);

/* CFL time step dt = cfl / max_zones sum_d c^d / dx_d from zone-centred fast-magnetosonic speeds c^d, for the
 * first step (the step is set by the signal crossing time of the smallest zones; S22).
 * *dt is a HOST double.  KH_ENAN if a primitive or a zone's speed is not finite. */
int kh_estimate_dt(kh_grid* g, double* dt);

/* One full predictor-corrector step:
 *     P* = substep(P^n, P^n, dt/2);   P^{n+1} = substep(P^n, P*, dt)
 * each sub-step = reconstruction + LLF fluxes per direction (K2), Flux-CT (K3), geometric source +
 * conserved update + 1D_W inversion + floors (K4/K5), ghost fill (K7), fix-up of failed zones (K5b),
 * ghost fill; the corrector's face speeds give the next CFL step (K6).
 *   dt > 0   : use this step
 *   dt <= 0  : use the device-resident dt_next of the previous step (no host round trip); KH_EINVAL
 *              before the first completed step of the grid
 *   dt_next  : HOST pointer receiving min(cfl * min_zones dt_zone, dt_growth_max * dt), or NULL to
 *              return without synchronising (the value stays on the device for the next dt <= 0 call)
 * KH_ENAN (with dt_next given): a zone's CFL rate of this step was not finite; dt_next is untouched.
 * The step replays a CUDA graph; if the stream cannot be captured the same kernels are launched directly. */
int kh_step(kh_grid* g, double dt, double* dt_next);

/* max |div B| of the corner-centred divergence that Flux-CT preserves.  HOST double. */
int kh_divB(kh_grid* g, double* max_abs);

/* The same divergence for callers that cannot allocate (code under CUDA-graph capture, serving loops, harnesses that forbid
 * cudaMalloc): no grid handle, no cudaMalloc / cudaFree / allocating library call, no synchronisation -- a memset node and one
 * kernel on `cuda_stream` (NULL: the legacy default stream).  The reduction's scratch is a static device array of
 * KH_NOALLOC_SCRATCH_BYTES that every GPU loading the library holds until exit; its address is looked up once per device on
 * the first call made with that device current (make one call before starting a capture).
 *   B        DEVICE, the field B^1..B^3 in the padded layout of kh_get_prims(with_ghosts = 1): [3][n3+6][n2+6][n1+6]
 *            (the last three components of that array); read only, owned by the caller;
 *   gdet     DEVICE, sqrt(-g) at zone centres as kh_get_geom(loc = 0) returns it, [n2+6][n1+6]; NULL = 1 (Minkowski);
 *   dx1..3   zone sizes (> 0);  lower_mask  bit d-1 set: the corners on the lower boundary plane of direction d count
 *            (their ghost zones hold data: periodic images or a neighbouring block's zones) -- kh_divB's own rule;
 *   max_abs  DEVICE, one double, written by the kernel: valid once the stream has reached it (+inf if a corner is NaN).
 * Errors: KH_EINVAL (NULL B / max_abs, sizes < 1, dx <= 0), KH_ESIZE when the corner count exceeds KH_NOALLOC_MAX_CORNERS
 * (nothing is enqueued), KH_ECUDA.  Every call shares the one scratch array per device: calls that overlap on the GPU (two
 * streams, two threads) race; calls ordered on one stream do not. */
#define KH_NOALLOC_MAX_CORNERS 16777216LL                       /* 65536 blocks of 256 corners: a 256^3 block fits */
#define KH_NOALLOC_SCRATCH_BYTES (8 * (32 + KH_NOALLOC_MAX_CORNERS / 256))
int kh_divB_noalloc(const double* B, const double* gdet, int n1, int n2, int n3, double dx1, double dx2, double dx3, int lower_mask,
                    double* max_abs, void* cuda_stream);

/* Number of zones with pflag != 0 and with fflag != 0 in the last sub-step (HOST ints; may be NULL). */
int kh_count_flags(kh_grid* g, long long* n_pflag, long long* n_fflag);

/* ---- several blocks on one device ("HARM requires two synchronizations") ----
 * A mesh block may be cut into several kh_grids along any direction.  A side whose neighbour is another block is created
 * with KH_BC_BLOCK; kh_link_blocks(lo, hi, dir) declares that `hi` continues `lo` across lo's upper dir-side (dir = 1..3;
 * both sides must be KH_BC_BLOCK, the transverse sizes, zone sizes, the stream and every option must agree; a periodic
 * direction cut in two is closed by a second link (hi, lo)).  Restrictions: fofc = 0, KH_B_FLUX_CT, KH_EMF_ARITHMETIC;
 * in FMKS cut along x2 or x3 (the map's x1 origin is a block's own xmin[0]).
 * kh_exchange_halos(blocks, n) packs the 3 layers next to every linked side (8 primitives + the inversion flag, over the full
 * padded transverse extent) into that side's message buffer and unpacks it into the neighbour's ghost layers -- on one
 * device the neighbour reads the buffer directly; the buffer is what an inter-GPU transport would send.  Call it after
 * loading primitives into linked blocks.
 * kh_step_blocks steps all n blocks (n <= 16) by dt together: per sub-step every block computes fluxes, EMFs, update and its
 * own boundary fills; halos are exchanged; every block repairs its failed zones (reading the neighbour's flags and values
 * through the halo); halos are exchanged again -- the two synchronisations of P:317 -- and dt_next is the minimum over the
 * blocks (one scalar reduction).  dt <= 0 and dt_next as for kh_step.  The result equals the single-block step bit for bit. */
int kh_link_blocks(kh_grid* lo, kh_grid* hi, int dir);
int kh_exchange_halos(kh_grid* const* blocks, int n);
int kh_step_blocks(kh_grid* const* blocks, int n, double dt, double* dt_next);

/* ---- stage access (tests / debugging) ---- */
/* Geometry tables over (j,i) with ghosts, [(n2+6)*(n1+6)] points: gcov/gcon as 16 doubles per point
 * (row-major 4x4), gdet and alpha one per point.  Any pointer may be NULL. */
int kh_get_geom(kh_grid* g, int loc, double* gcov16, double* gcon16, double* gdet, double* alpha, int mem);
/* Connection Gamma^lam_{mu nu} at centres: 64 doubles per (j,i) point, [lam][mu][nu]. */
int kh_get_conn(kh_grid* g, double* conn64, int mem);
/* LLF face fluxes of direction dir (1..3) of the last sub-step, with ghosts [8][nt], index = lower
 * face of the zone; hydro components as used by the update, B components replaced by their Flux-CT
 * values (computed from the edge EMFs); ctop [nt].  Entries outside the computed face range are 0. */
int kh_get_flux(kh_grid* g, int dir, double* F, double* ctop, int mem);
/* Face-centred CT (kh_params.transport = KH_B_FACE_CT).  Phi^d = sqrt(-g) B^d on the lower d-face of each zone, three
 * arrays with ghosts [nt] (faces i_d in [0, N_d] with interior transverse indices are used, the rest ignored).
 * kh_set_face_B also sets the zone-centred field of the current state to the mean of each zone's two face values over
 * sqrt(-g) and fills its ghosts: call it AFTER kh_set_prims; kh_step returns KH_EINVAL on a face-CT grid until it has been
 * called.  kh_divB_face: max over interior zones of
 * |sum_d (Phi^d(upper) - Phi^d(lower))/dx_d|, which the transport keeps at its initial value to round-off. */
int kh_set_face_B(kh_grid* g, const double* f1, const double* f2, const double* f3, int mem);
int kh_get_face_B(kh_grid* g, double* f1, double* f2, double* f3, int mem);
int kh_divB_face(kh_grid* g, double* max_abs);
/* Edge EMFs of the last sub-step, with ghosts [nt], index = lower edge of the zone. */
int kh_get_emf(kh_grid* g, int dir, double* emf, int mem);
/* Run the fix-up (K5b) + floors + refresh of the fixed zones' ghost images on the current primitives for a caller-supplied flag array
 * (int32, with ghosts [nt]); test hook for hand-built neighbourhoods. */
int kh_debug_fixup(kh_grid* g, const int* pflag_with_ghosts, int mem);
/* Run only the predictor sub-step P* = substep(P^n, P^n, dt/2) and make P* the current state (test hook:
 * exposes the intermediate state and the predictor's fluxes / flags to the stage getters). */
int kh_debug_predictor(kh_grid* g, double dt);
/* Number of kernel launches enqueued by this grid since creation. */
long long kh_launch_count(const kh_grid* g);
/* Enable/disable CUDA-graph replay of kh_step (default on); the first step after a change captures. */
int kh_set_graph(kh_grid* g, int enable);
/* Per-kernel device timing.  While enabled, kh_step replays a second, instrumented CUDA graph of the step whose launch
 * groups are bracketed by event-record nodes, and reads them out (synchronising) after every step, so the kernels are
 * timed running exactly as in the product path; with graph replay off (kh_set_graph(g, 0)) the kernels are enqueued
 * directly between event pairs.  A launch group is one kernel, except: the three flux directions of a sub-step, which run
 * concurrently, are ONE group reported under KH_K_FLUX1 (KH_K_FLUX2 / 3 then stay empty); the fix-up's two kernels are one
 * group.  kh_get_profile returns, per kind (KH_K_*), the summed device milliseconds and the number of groups since
 * kh_set_profile(g, 1).  ms and count are HOST arrays of KH_K_COUNT entries.  Used by bench.py for the per-kernel roofline;
 * headline throughput is always measured with profiling off. */
enum { KH_K_FLUX1 = 0, KH_K_FLUX2 = 1, KH_K_FLUX3 = 2, KH_K_EMF = 3, KH_K_UPDATE = 4, KH_K_FILL = 5, KH_K_FIXUP = 6,
       KH_K_FOFC = 7 /* mask + re-flux of the first-order flux correction */, KH_K_COUNT = 8 };
int kh_set_profile(kh_grid* g, int enable);
int kh_get_profile(kh_grid* g, double* ms, long long* count);
/* Stand-alone DFMA-chain micro-benchmark: returns achieved fp64 TFLOP/s on the current device
 * (HOST double) -- the measured fp64 peak used as an ALU roofline denominator by bench.py. */
int kh_measure_fp64_peak(double* tflops, double* sm_mhz_est);

const char* kh_strerror(int code);
const char* kh_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif

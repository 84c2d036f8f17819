/* kho.h -- C interface of the CPU ORACLE of the HARM/KHARMA ideal-GRMHD step.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, header,
 * table or helper with the CUDA path under paper_2408_01361_b200/ (which has its own
 * include/kharm.h); the struct below is deliberately a separate definition.
 *
 * What it computes: one explicit second-order predictor-corrector ideal-GRMHD update of a
 * uniform logically-Cartesian block in a stationary metric, fp64, single thread, triple loops.
 * PAPER.md prints only eq. 1.1 (T^{mu nu}, line 347) of the scheme; everything else is the
 * published mathematics of the schemes it cites at PAPER.md line 243 (HARM, modified velocity,
 * 1D_W inversion, Flux-CT), line 253 (MC, WENO5), line 111 (FMKS) -- see DESIGN.md section
 * "Readings" (S1..S23) for every point the paper leaves open.
 *
 * All pointers are HOST pointers. Arrays are fp64, SoA [var][k][j][i], x1 (i) fastest.
 * "with ghosts" arrays have NG = 3 layers per side in all three directions.
 */
#ifndef KHO_H
#define KHO_H
#ifdef __cplusplus
extern "C" {
#endif

enum { KHO_MINKOWSKI = 0, KHO_KS = 1, KHO_FMKS = 2 };
enum { KHO_BC_PERIODIC = 0, KHO_BC_OUTFLOW = 1, KHO_BC_POLAR = 2, KHO_BC_FIXED = 3 };
enum { KHO_RECON_MC = 0, KHO_RECON_WENO5 = 1 };
enum { KHO_INV_1DW = 0, KHO_INV_KASTAUN = 1 };
enum { KHO_FRAME_FLUID = 0, KHO_FRAME_DRIFT = 1, KHO_FRAME_NORMAL = 2 };
enum { KHO_B_FLUX_CT = 0, KHO_B_FACE_CT = 1 };
enum { KHO_EMF_ARITHMETIC = 0, KHO_EMF_UPWIND = 1, KHO_EMF_CENTRED = 2 };
enum { KHO_LOC_CENT = 0, KHO_LOC_FACE1 = 1, KHO_LOC_FACE2 = 2, KHO_LOC_FACE3 = 3 };

typedef struct {
  int coords;
  double a;                                        /* BH spin (KS / FMKS)                 */
  double hslope, poly_xt, poly_alpha, mks_smooth;  /* FMKS map parameters                 */
  int n1, n2, n3;                                  /* interior zones                      */
  double xmin[3], xmax[3];                         /* native bounds of the interior       */
  int bc[6];                                       /* x1lo x1hi x2lo x2hi x3lo x3hi       */
  double gamma, cfl;
  int recon;
  double rho_min, u_min, r_char, bsq_over_rho_max, bsq_over_u_max, u_over_rho_max, gamma_max;
  double dt_growth_max;
  int inverter;                                    /* KHO_INV_1DW | KHO_INV_KASTAUN (NEXT-2) */
  int fofc;                                        /* 1: first-order flux correction (NEXT-3) */
  int floor_frame;                                 /* KHO_FRAME_FLUID | _DRIFT | _NORMAL (NEXT-4) */
  int transport;                                   /* KHO_B_FLUX_CT | KHO_B_FACE_CT (NEXT-1) */
  int emf;                                         /* KHO_EMF_ARITHMETIC | KHO_EMF_UPWIND | KHO_EMF_CENTRED (NEXT-1) */
} kho_params;

typedef struct kho_grid kho_grid;

/* ---- grid-level calls (mirror the product's kh_* calls) ---- */
int kho_grid_create(const kho_params* p, kho_grid** out);
int kho_grid_destroy(kho_grid* g);
int kho_set_prims(kho_grid* g, const double* p, int with_ghosts);
int kho_get_prims(kho_grid* g, double* p, int with_ghosts);
int kho_get_cons(kho_grid* g, double* u);                 /* interior [8][n3][n2][n1]     */
int kho_get_flags(kho_grid* g, int* pflag, int* fflag);   /* interior, last sub-step      */
int kho_estimate_dt(kho_grid* g, double* dt);
int kho_step(kho_grid* g, double dt, double* dt_next);
int kho_divB(kho_grid* g, double* max_abs);
/* face-centred CT (NEXT-1): Phi^d = sqrt(-g) B^d on the lower d-face of each zone, with ghosts [nt] each (faces
 * i_d in [0, N_d], transverse interior are used); setting it also sets the zone-centred B of the current state */
int kho_set_face_B(kho_grid* g, const double* f1, const double* f2, const double* f3);
int kho_get_face_B(kho_grid* g, double* f1, double* f2, double* f3);
int kho_divB_face(kho_grid* g, double* max_abs);   /* max |sum_d (Phi^d(+1) - Phi^d)/dx_d| over interior zones */
/* stage access for tests: fluxes after Flux-CT of the LAST sub-step, with ghosts [8][nt]; ctop [nt] */
int kho_get_flux(kho_grid* g, int dir, double* F, double* ctop);
int kho_get_emf(kho_grid* g, int dir, double* emf);
/* geometry tables: loc in KHO_LOC_*, arrays over (j,i) with ghosts: [(n2+6)][(n1+6)] rows     */
int kho_get_geom(kho_grid* g, int loc, double* gcov16, double* gcon16, double* gdet, double* alpha);
int kho_get_conn(kho_grid* g, double* conn64);            /* [(n2+6)(n1+6)][lam][mu][nu]  */
int kho_fill_ghosts(kho_grid* g);
/* test hook: C9 fix-up (+ floors) of the current primitives for a caller-supplied pflag array [nt] */
int kho_debug_fixup(kho_grid* g, const int* pflag_with_ghosts);
/* test hook (NEXT-1): high-order fluxes of the current primitives and the edge EMFs of the configured kind; leaves the RAW
 * face fluxes (no Flux-CT rewrite) for kho_get_flux and the EMFs for kho_get_emf */
int kho_debug_emf(kho_grid* g);
/* test hook (NEXT-3): high-order fluxes of the current primitives, then the first-order flux correction for a caller-
 * supplied zone mask [nt] (its ghosts are filled like pflag); leaves the RAW fluxes (no Flux-CT) for kho_get_flux */
int kho_debug_fofc(kho_grid* g, const int* mask_with_ghosts);
/* test hook: predictor sub-step only; P* becomes the current state */
int kho_debug_predictor(kho_grid* g, double dt);

/* ---- point-wise pieces, exposed so tests can pin them one by one ---- */
/* embedding coordinates (r, theta, phi) or (x,y,z) of a native point */
void kho_embed(const kho_params* p, const double X[3], double emb[3]);
/* covariant metric, inverse, sqrt(-g), lapse at a native point (x3 irrelevant) */
void kho_metric(const kho_params* p, double x1, double x2, double gcov[16], double gcon[16],
                double* gdet, double* alpha);
/* connection Gamma^lam_{mu nu} by exact (forward-mode) differentiation of gcov */
void kho_conn(const kho_params* p, double x1, double x2, double conn[64]);
/* same by centred finite differences of step h (cross-check only) */
void kho_conn_fd(const kho_params* p, double x1, double x2, double h, double conn[64]);
/* 4-vectors of a primitive state: out = ucon[4] ucov[4] bcon[4] bcov[4] bsq (17 doubles) */
void kho_fourvec(const double gcov[16], const double gcon[16], const double P[8], double out[17]);
/* dir = 0: conserved U; dir = 1..3: flux F^dir */
void kho_prim_to_flux(const double gcov[16], const double gcon[16], double gdet, const double P[8],
                      double gamma, int dir, double F[8]);
/* mixed stress tensor T^mu_nu, eq. 1.1 with one index lowered; T[mu*4+nu] */
void kho_stress(const double gcov[16], const double gcon[16], const double P[8], double gamma,
                double T[16]);
void kho_vchar(const double gcov[16], const double gcon[16], const double P[8], double gamma,
               int dir, double* vmax, double* vmin);
/* reconstruction of one variable on a 5-point stencil q[-2..2] -> zone's left/right face value */
void kho_recon(int recon, const double q[5], double* left, double* right);
void kho_llf(const double gcov[16], const double gcon[16], double gdet, const double PL[8],
             const double PR[8], double gamma, int dir, double F[8], double* ctop);
void kho_source(const double gcov[16], const double gcon[16], double gdet, const double conn[64],
                const double P[8], double gamma, double S[8]);
/* Test hook: Qt^2 = g_ij Qt^i Qt^j of the projected momentum exactly as kho_u2p forms it from the covariant Q_mu (DESIGN S16) */
double kho_qtsq(const double gcov[16], const double gcon[16], double alpha, const double Qcov[4]);
/* U -> P (1D_W); returns the flag (0 = ok). Pout holds guess hydro prims on failure. */
int kho_u2p(const double gcov[16], const double gcon[16], double gdet, const double U[8],
            const double Pguess[8], double gamma, double Pout[8]);
/* U -> P by the bracketed root find of Kastaun et al.; same flag convention */
int kho_u2p_kastaun(const double gcov[16], const double gcon[16], double gdet, const double U[8],
                    const double Pguess[8], double gamma, double Pout[8]);
/* floors at a native point; returns fflag bits */
int kho_floors(const kho_params* p, const double gcov[16], const double gcon[16], double x1,
               double x2, double P[8]);
/* Flux-CT on caller-supplied face fluxes (with ghosts, [8][nt] each); rewrites the B components */
int kho_flux_ct_arrays(const kho_params* p, double* F1, double* F2, double* F3);

const char* kho_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif

/* hzo.h -- C ABI of the CPU ORACLE for the HORIZON per-substep GRMHD update.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load this library.
 * It shares no source, header, table or helper with the CUDA path
 * (paper_1102_5202_b200/csrc, include/hz.h) and neither includes the other.
 *
 * What it computes: one method-of-lines Runge-Kutta substep of the finite-volume
 * GRMHD scheme the paper describes in PAPER.md:74-80 (section 2.2) with the named
 * ingredients of PAPER.md:128 (section 3.2): HLLE fluxes, TVD reconstruction with
 * the MC limiter, Newton-Raphson primitive recovery, third-order Runge-Kutta,
 * hyperbolic divergence cleaning; continuum system PAPER.md:44-58 (eqs. 1-2).
 * The discrete formulas the paper does not print are the readings O1-O10 /
 * R1-R22 of SURVEY.md section 8(c), restated in DESIGN.md.
 *
 * All pointers are HOST pointers to double.  Field arrays are interior-only,
 * nx*ny*nz per plane, x fastest, planes concatenated.
 *
 * Point ordering conventions
 *   prim9 : rho, ut^x, ut^y, ut^z, p, B^x, B^y, B^z, psi      (ut^i = W v^i)
 *   cons9 : D, S_x, S_y, S_z, tau, B^x, B^y, B^z, psi          (NOT densitised)
 *   met10 : alpha, beta^x, beta^y, beta^z, g_xx, g_xy, g_xz, g_yy, g_yz, g_zz
 *   prim8 (API): rho, v^x, v^y, v^z, p, B^x, B^y, B^z         (v^i Eulerian 3-velocity)
 */
#ifndef HZO_H
#define HZO_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct hzo_ctx hzo_ctx;

enum { HZO_BC_PERIODIC = 0, HZO_BC_OUTFLOW = 1 };
enum { HZO_OK = 0, HZO_EINVAL = -1, HZO_ENOMEM = -2, HZO_ESTATE = -4 };

typedef struct { int nx, ny, nz; double dx, dy, dz; int bc[3]; } hzo_grid;

typedef struct {
  double gamma_ad;         /* ideal-gas Gamma                                        */
  double rho_atm, p_atm;   /* atmosphere values                                      */
  double atm_tol;          /* reset if rho < rho_atm*(1+atm_tol)                     */
  int    cleaning;         /* 0: psi frozen at 0; 1: hyperbolic cleaning on          */
  double kappa;            /* cleaning damping rate                                  */
  int    c2p_maxit;        /* Newton iteration cap                                   */
  double c2p_tol;          /* |dZ| <= tol*Z                                          */
  int    c2p_scheme;       /* 0: Newton on Z (O8); 1: Newton on (Z, v^2) (O8b)       */
  int    energy_var;       /* 0: evolve sqrt(gamma) tau (R1); 1: the paper's          */
                           /* -sqrt(-g) T^t_t (R1b): slot 4 of U, source-free        */
  int    recon;            /* 0: MC-limited linear (O4); 1: PPM (O4b), 3 ghost layers */
} hzo_params;

typedef struct {
  double sumD, sumSx, sumSy, sumSz, sumTau;  /* sum over interior of sqrt(gamma)*(..)*dx*dy*dz */
  double sumBx, sumBy, sumBz, sumPsi;
  double divB_max, divB_L1;                  /* centred div(sqrt(gamma) B)/sqrt(gamma)          */
  double max_speed_over_dx;                  /* max_d max(|lam+|,|lam-|)/dx_d                   */
  long long c2p_fail, atm_reset, p_floor;    /* cumulative counters since set_primitives        */
  int c2p_maxit_seen;
} hzo_diag;

/* ---- point functions (pins call these one state at a time) --------------------- */
int    hzo_prim2con_point(const double* prim9, const double* met10, double gamma_ad, double* cons9);
/* returns 0 converged, 1 failed.  Zguess <= 0 selects the built-in guess.              */
int    hzo_con2prim_point(const double* cons9, const double* met10, const hzo_params* par,
                          double Zguess, double* prim9, int* iters);
double hzo_c2p_residual_point(double Z, const double* cons9, const double* met10, double gamma_ad);
/* coordinate flux (alpha*F^d for D,S,tau; the O2 rows for B,psi), NOT times sqrt(gamma) */
int    hzo_flux_point(int d, const double* prim9, const double* met10, double gamma_ad,
                      int cleaning, double* flux9);
int    hzo_wavespeed_point(int d, const double* prim9, const double* met10, double gamma_ad,
                           int cleaning, double* lam_minus_plus);
double hzo_mc_slope(double qm, double q0, double qp);
void hzo_ppm_edges(const double* q5, double* aL, double* aR);
/* HLLE flux Phi = sqrt(gamma_f) * Fhat through one face with face metric met10 */
int    hzo_hlle_point(int d, const double* primL, const double* primR, const double* met10,
                      double gamma_ad, int cleaning, double* phi9);
/* fluid source alpha*sqrt(gamma)*Sigma for (S_x,S_y,S_z,tau) given metric derivatives
 * dmet30[j*10 + c] = d_j met10[c].                                                      */
int    hzo_source_point(const double* prim9, const double* met10, const double* dmet30,
                        double gamma_ad, double* src4);

/* ---- grid API (mirrors the hz_* boundary of include/hz.h) ----------------------- */
int  hzo_default_params(hzo_params*);
int  hzo_create(const hzo_grid*, const hzo_params*, hzo_ctx** out);
int  hzo_destroy(hzo_ctx*);
int  hzo_set_metric(hzo_ctx*, const double* alpha, const double* beta3, const double* gamma6);
int  hzo_set_primitives(hzo_ctx*, const double* prim8);
int  hzo_step(hzo_ctx*, double dt, int n);          /* n full RK3 steps                        */
int  hzo_substeps(hzo_ctx*, double dt, int nsub);    /* nsub RK substeps, continuing the stage  */
int  hzo_get_primitives(hzo_ctx*, double* prim8);
int  hzo_get_psi(hzo_ctx*, double* psi);
int  hzo_get_conserved(hzo_ctx*, double* cons9);     /* densitised sqrt(gamma)*(D,S,tau,B,psi)  */
int  hzo_get_rhs(hzo_ctx*, double* rhs9);            /* L(U) for the current primitives         */
int  hzo_diagnostics(hzo_ctx*, hzo_diag*);
/* test accessors, no arithmetic: set the cleaning scalar psi (interior planes; U and ghosts follow), read
 * the padded extents (cells and ghost layers per axis) and one padded array (which: 0 primitives, 1 metric;
 * x fastest, N[0]*N[1]*N[2] values) */
int  hzo_set_psi(hzo_ctx*, const double* psi);
int  hzo_padded_extent(const hzo_ctx*, int* N3, int* g3);
int  hzo_get_padded(hzo_ctx*, int which, int field, double* out);
int  hzo_num_threads(void);
const char* hzo_strerror(int);

#ifdef __cplusplus
}
#endif
#endif

/* oracle/oracle.h — C interface of the CPU test oracle (TEST INFRASTRUCTURE, NOT THE PRODUCT).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load
 * liboracle.so.  The product library (include/mhd.h, libmhd.so) neither includes this file nor links it.
 * All pointers are HOST pointers; all field arrays are N^3 doubles laid out [z][y][x] (x fastest).
 * Functions return 0 on success, a negative number on error (orc_last_error() gives the text).
 */
#ifndef ORACLE_H
#define ORACLE_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct orc_ctx orc_ctx;

typedef struct {
    double t;
    long long step;
    double ke, me, ie, mass, mom[3], etot, max_divb, rho_min, p_min;
} orc_diag;

/* precision: 0 = double arithmetic, 1 = long double arithmetic (inputs/outputs stay double). */
int orc_create(orc_ctx **out, int N, double L, double gamma, double mu, double eta, double dt, int precision);
int orc_destroy(orc_ctx *c);
const char *orc_last_error(void);
void orc_set_threads(int n);               /* OpenMP threads used by the pencil loops (0 = default)  */
int orc_get_threads(void);
int orc_use_direct_dft(orc_ctx *c, int on); /* substitute the O(N^6) DFT for the FFT (pin P13)        */

/* equation-set variants (Eq. 5/18 barotropic closure, Eq. 18 + L215 ABC forcing, L199/L205 switched-off
 * equations): cs2 > 0 selects P = cs2*rho; f0, kf = forcing amplitude and integer mode; evolve bit 0 = Eq. 17-18 (+E),
 * bit 1 = Eq. 19 */
int orc_set_variant(orc_ctx *c, double cs2, double f0, int kf, int evolve);
int orc_set_stress(orc_ctx *c, int on);   /* 1: viscous terms of Eq. 11-12 (2 nu rho S, nu = mu) instead of mu lap u */
int orc_set_integrator(orc_ctx *c, int integrator);   /* 0 AB2 (default), 1 RK4, 2 predictor-corrector (Heun); L25, L39 */
int orc_set_fields(orc_ctx *c, int kind, const double *const f[8]);  /* 0 conservative, 1 primitive  */
int orc_get_fields(orc_ctx *c, int kind, double *const out[8]);
int orc_rhs(orc_ctx *c, double *const out[8]);                       /* dU/dt of the current state    */
int orc_rhs_scales(orc_ctx *c, double *const out[8], double phi[8], double dsc[8]);
int orc_step(orc_ctx *c, int nsteps);
int orc_nspec(orc_ctx *c);
int orc_diagnostics(orc_ctx *c, orc_diag *d, double *spec_kin, double *spec_mag, int nspec);

/* operator family O1 on one field: op 0,1,2 = d/dx,d/dy,d/dz; 3 = Laplacian; 4 = dealias projection */
int orc_apply(orc_ctx *c, int op, const double *in, double *out);

/* transforms O0 on interleaved (re,im) complex N^3 arrays; sign -1 forward (unnormalised), +1 inverse (1/N^3) */
int orc_fft3(int N, int sign, int precision, const double *in, double *out);
int orc_dft3_direct(int N, int sign, int precision, const double *in, double *out);

/* ---- tracer particles, Sec. VI (L229-275), oracle/tracers_oracle.hpp ---------------------------------
 * Stand-alone pieces (fp64): CIC interpolation (Eq. 20) of nf grid fields to np positions; nsteps Boris pushes
 * (Eq. 21-22) in a FROZEN grid field B[3].  pos / vel are 3 arrays of np doubles (x, y, z components). */
int orc_cic(int N, double L, int nf, const double *const g[], long long np, const double *const pos[3],
            double *const out[]);
int orc_tracers_push(int N, double L, double dt, const double *const B[3], long long np, double *const pos[3],
                     double *const vel[3], int nsteps);
/* Tracers attached to a solver: orc_step() then pushes them once per step with the B of the state at the START of
 * the step (t_n), before the fields advance.  vel == NULL: initial velocity = CIC interpolation of u = m/rho. */
int orc_tracers_set(orc_ctx *c, long long np, const double *const pos[3], const double *const vel[3]);
int orc_tracers_get(orc_ctx *c, double *const pos[3], double *const vel[3]);

#ifdef __cplusplus
}
#endif
#endif

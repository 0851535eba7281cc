// kernels.h — host-side declarations of the kernel launchers of libmhd (internal; the public ABI is include/mhd.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mhd {

typedef double2 cd;
constexpr int MAXF = 16;   // largest batch of fields one launch handles

// Physical constants of one context, passed by value to the point-wise kernels.
struct Phys {
    double k0;       // 2*pi/L : wavenumber of integer mode 1
    double gamma, mu, eta;
};

// ---- strided (y / z) complex passes on [kz][ky][kx] half-spectrum arrays with row pitch `hx` ------------
struct StridedArgs {
    const cd* in[MAXF];
    cd* out[MAXF];
    const cd* tw;          // exp(-2 pi i m / N), m < N
    long long row_stride;  // complex elements between consecutive points of the transformed axis
    long long outer_stride;// complex elements between consecutive outer indices
    int nchunks;           // column chunks (of C columns) to process
    int ncols;             // valid columns (guards the last chunk)
    int n_outer;           // number of outer indices processed
    int outer_split;       // outer index o maps to o (o < split) or o + outer_skip
    int outer_skip;
    int kc;                // 2/3 cut-off
    int in_pruned;         // rows outside the mask are not read (taken as zero)
    int out_pruned;        // rows outside the mask are not written
    int nfields;
};
// dir = -1 forward, +1 inverse (unnormalised both ways)
void launch_strided(int N, int dir, const StridedArgs& a, cudaStream_t st);

// ---- x passes ----------------------------------------------------------------------------------------------
struct XArgs {
    const double* real_in[MAXF];   // r2c input lines  (N doubles per line)
    double* real_out[MAXF];        // c2r output lines
    const cd* spec_in[MAXF];       // c2r input  (N/2 complex per line, Nyquist dropped)
    cd* spec_out[MAXF];            // r2c output
    cd* nyq_out[MAXF];             // r2c: optional Nyquist column, [row][8] complex with column 0 used (or null)
    const cd* tw;                  // exp(-2 pi i m / N)
    long long nlines;              // lines per field (N*N)
    int kmax;                      // highest kx read (c2r) / written (r2c): N/2-1 unpruned, kc pruned
    int nfields;
    double scale;                  // c2r: factor applied to the output (1/N^3)
};
void launch_x_r2c(int N, const XArgs& a, cudaStream_t st);
void launch_x_c2r(int N, const XArgs& a, cudaStream_t st);

// fused real-axis sweep: c2r of 11 fields (8 state + 3 current), flux products, r2c of 16 product fields
struct FusedXArgs {
    const cd* in[11];     // rho, mx, my, mz, E, Bx, By, Bz, Jx, Jy, Jz  (half-spectrum after the y pass)
    cd* out[16];          // Txx,Txy,Txz,Tyy,Tyz,Tzz, FEx,FEy,FEz, ex,ey,ez, ux,uy,uz, q
    const cd* tw;
    long long nlines;
    int kmax_in, kmax_out;
    double scale;
    Phys ph;
};
void launch_x_fused(int N, const FusedXArgs& a, cudaStream_t st);
// second-generation fused sweep (kernels_xfused2.cu): N = 128, 256, 512
bool x_fused2_supported(int N);
void launch_x_fused2(int N, const FusedXArgs& a, cudaStream_t st);   // a.tw = the lane-contiguous tables below
int x_fused2_table_entries(int N);
void launch_x_fused2_tables(int N, cd* tab, cudaStream_t st);

// ---- point-wise kernels -------------------------------------------------------------------------------
// real space: 11 fields in -> 16 product fields out (same slot order as FusedXArgs)
void launch_flux_real(long long n, const double* const in[11], double* const out[16], Phys ph, cudaStream_t st);
// primitive <-> conservative, in place on 8 real fields
void launch_prim_to_cons(long long n, double* const f[8], double gamma, cudaStream_t st);
void launch_cons_to_prim(long long n, double* const f[8], double gamma, cudaStream_t st);

struct SpecGeom {
    int N, hx, kc;     // hx = row pitch in complex elements (N/2)
    int pruned;        // visit only modes inside the mask (1) or all stored modes (0; masked ones get zero)
};
// J^ = M i k x B^
void launch_build_current(const SpecGeom& g, const cd* const B[3], cd* const J[3], Phys ph, cudaStream_t st);
// R^ from the 16 transformed product fields and the state; mode 0: write R^ to rout only;
// mode 1: Euler update U += dt R, Rold = R; mode 2: AB2 update U += dt(1.5 R - 0.5 Rold), Rold = R
void launch_assemble(const SpecGeom& g, const cd* const prod[16], cd* const U[8], cd* const Rold[8],
                     cd* const rout[8], int mode, double dt, Phys ph, cudaStream_t st);
// generic linear update on masked modes: y[f] = a*y[f] + b*x[f] ... used by RK4 / predictor-corrector
void launch_axpby(const SpecGeom& g, int nf, double a, cd* const y[], double b, const cd* const x[], cudaStream_t st);
void launch_copy_masked(const SpecGeom& g, int nf, cd* const dst[], const cd* const src[], cudaStream_t st);
// div^ = M i k . B^
void launch_divergence(const SpecGeom& g, const cd* const B[3], cd* out, Phys ph, cudaStream_t st);
// zero everything outside the mask (and optionally everything) of nf spectral arrays
void launch_zero_outside_mask(const SpecGeom& g, int nf, cd* const f[], cudaStream_t st);

// ---- diagnostics ----------------------------------------------------------------------------------------
// block partials -> out[0..11]: ke, me, ie, mass, momx, momy, momz, etot (sums), rho_min, p_min; deterministic
void launch_diag_reduce(long long n, const double* const U[8], double gamma, double* scratch, double* out,
                        cudaStream_t st);
void launch_absmax(long long n, const double* f, double* scratch, double* out, cudaStream_t st);
// w_c = m_c / sqrt(rho)
void launch_sqrt_rho_u(long long n, const double* const U[8], double* const w[3], cudaStream_t st);
// shell spectrum of 3 components: S[K] += weight * 1/2 |w^|^2 / N^6 ; deterministic two-stage reduction
void launch_shell_spectrum(int N, const cd* const spec[3], const cd* const nyq[3], double* scratch, double* out,
                           int nspec, cudaStream_t st);
int diag_scratch_doubles(int nspec);

void launch_twiddle_table(int N, cd* tw, cudaStream_t st);

}  // namespace mhd

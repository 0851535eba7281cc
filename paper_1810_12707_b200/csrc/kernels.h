// kernels.h — host-side declarations of the kernel launchers of libmhd (internal; the public ABI is include/mhd.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mhd {

typedef double2 cd;
constexpr int MAXF = 16;   // largest batch of fields one launch handles

// Opt-in to more than 48 KB of dynamic shared memory (and, for the cluster kernels, to a non-portable cluster size), once
// per kernel instantiation AND per device (the attributes are per-device properties of the function: a process that drives
// several GPUs must set them on each of them).
// The cache is keyed by the kernel's ADDRESS (all instantiations of one template share the pointer type K, so a
// function-local static keyed by K alone would configure only the first of them).  Check, cudaFuncSetAttribute and the
// record happen under ONE lock, and (kernel, device) is recorded only when every attribute was set: a second host thread
// cannot launch before the opt-in has landed, and a failed opt-in is retried by the next launch and reported — the
// cudaError_t stays in the runtime's last-error slot for check_cuda(), which also names the failing step
// (kernel_config_error()).
cudaError_t configure_kernel(const void* kern, size_t smem, bool nonportable_cluster = false);      // mhd_api.cu
const char* kernel_config_error();      // description of this thread's last failed configure_kernel ("" = none); clears it
template <class K> inline void ensure_dynamic_smem(K kern, size_t smem) {
    configure_kernel(reinterpret_cast<const void*>(kern), smem);
}

// Physical constants of one context, passed by value to the point-wise kernels.
struct Phys {
    double k0;       // 2*pi/L : wavenumber of integer mode 1
    double gamma, mu, eta;
    // equation-set variants (Eq. 5/18, L192, L199, L205, L215)
    double cs2;      // > 0: barotropic closure P = cs2 * rho, the energy equation is not evolved
    double f0;       // amplitude of the ABC forcing rho f (0 = unforced)
    int kf;          // its integer mode number
    int evolve;      // bit 0: Eq. 17-18 (+ energy) evolve; bit 1: Eq. 19 evolves
};

// ---- strided (y / z) complex passes on half-spectrum arrays ------------------------------------------------
// The transformed axis ("rows") and one outer axis are addressed by strides, so the same kernel serves the
// in-place in-core sweeps on [kz][ky][kx] arrays (pitch N/2) and the bricks / slabs of the out-of-core
// pipeline (compact layouts, separate input and output views).
// Row storage modes: 0 = all N rows stored; 1 = all N rows stored, rows outside the 2/3 mask are not touched
// (read as zero / not written); 2 = compact: only the 2kc+1 rows inside the mask are stored, consecutively
// (row r <= kc at r, row r >= N-kc at r - (N - 2kc - 1)).
struct StridedArgs {
    const cd* in[MAXF];
    cd* out[MAXF];
    const cd* tw;          // exp(-2 pi i m / N), m < N
    long long in_row_stride, out_row_stride;      // complex elements between consecutive stored rows
    long long in_outer_stride, out_outer_stride;  // complex elements between consecutive outer indices
    int nchunks;           // (computed by the launcher from ncols and the columns per CTA)
    int ncols;             // valid columns (guards the last chunk)
    int n_outer;           // number of outer indices processed
    int outer_split;       // in-core: outer index o maps to o (o < split) or o + outer_skip
    int outer_skip;
    int kc;                // 2/3 cut-off
    int in_rows;           // row storage mode of the input (0, 1, 2)
    int out_rows;          // row storage mode of the output
    int nfields;
    int general;           // 0: in-core fast path (out strides = in strides, row modes 0/1); 1: general views
    // Fused current (sweep S1): fields f >= jfirst are not read from in[f]; they are built on load as
    // J^_c = M (i k x B^)_c from in[bfirst .. bfirst+2] (rows = kz, outer = ky, columns = kx).  jfirst < 0: off.
    int jfirst, bfirst;
    // Multi-GPU slab decomposition (general views only): output rows are owned by different ranks; row sr (stored index)
    // belongs to peer p with peer_lo[p] <= sr < peer_lo[p+1] and is written at out + peer_delta[p] (complex elements):
    // the same location inside that peer's workspace, reached through a peer mapping (NVLink P2P stores).  npeer = 0: off.
    int npeer;
    int peer_lo[9];
    long long peer_delta[8];
    int outer_compact;     // 1: outer index (+ outer_base) is a compact ky index; 0: a full array index
    int outer_base;
    double k0;             // 2 pi / L
};
// dir = -1 forward, +1 inverse (unnormalised both ways)
void launch_strided(int N, int dir, const StridedArgs& a, cudaStream_t st);

// The same in-core passes as a persistent, TMA-fed pipeline (kernels_strided_tma.cu): N = 128, 256, 512, arrays that are
// field buffers of the workspace (tensor maps are built over it at bind time), no fused current, no peer stores.
struct StridedTma {
    const void* maps = nullptr;    // 4 CUtensorMap: (rows = y | z) x (box rows = kc + 1 | N / 2), or null: not available
    const void* base = nullptr;    // first field buffer
    size_t stride_bytes = 0;       // distance between field buffers
    int nbuf = 0;                  // number of field buffers
    int sms = 0;                   // CTAs of the persistent grid (= multiprocessors of the device)
};
bool strided_tma_supported(int N);
bool strided_tma_build_maps(int N, void* base, size_t stride_bytes, int nbuf, void* maps_out);
bool launch_strided_tma(int N, int dir, const StridedArgs& a, const StridedTma& tm, cudaStream_t st);   // false: not eligible

// Sweep S5 as ONE launch (north_star (4): "the explicit time integrator fused into the last spectral
// pass"): the in-core forward z pass of the 16 product fields in thread-block clusters of 16 — one CTA per field of a
// (ky, kx tile) column — which keep the transformed rows in shared memory, meet at a cluster barrier and assemble R^
// (i k, -k^2, mask) and the explicit update from each other's tiles through distributed shared memory.
struct AssembleTail {
    cd* U[8];
    cd* Rold[8];
    cd* rout[8];           // mode 0 only
    int mode;              // as launch_assemble: 0 rout = R; 1 Euler update; 2 Adams-Bashforth 2 update
    double dt;
    Phys ph;
};
bool strided_assemble_supported(int N);
void launch_strided_assemble(int N, int fields_per_cta, const StridedArgs& a, const AssembleTail& z, cudaStream_t st);
int strided_assemble_max_clusters(int N, int fields_per_cta, const StridedArgs& a);   // occupancy query (bench / diagnostics)

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
    double* breal[3];     // optional (fused2 only): real-space Bx, By, Bz lines are also written here (tracers); or null
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
    // Compact bricks (out-of-core pipeline): the arrays hold only rows inside the mask.  Thread (ix, oy, oz) with
    // oy < ny, oz < 2kc+1 addresses "work" arrays at oz*wsz + oy*wsy + ix and "state" arrays at oz*ssz + oy*ssy + ix;
    // its ky mode follows from the compact index oy + y0.  compact = 0: both are the full [kz][ky][kx] index.
    int compact, y0, ny;
    long long wsy, wsz, ssy, ssz;
};
// J^ = M i k x B^
void launch_build_current(const SpecGeom& g, const cd* const B[3], cd* const J[3], Phys ph, cudaStream_t st);
// One stage of a multi-stage integrator in low-storage form (mode 3; RK4 and the predictor-corrector, Table I
// L39): with the stage slope R just assembled,  first: U0 <- U;  acc <- acc + b_acc R (first: b_acc R);  U <- U0 + c_next R;
// last stage instead: U <- U0 + acc + b_acc R.  One pass over the modes per stage, no separate linear-combination kernels.
struct StageUpdate {
    cd* U0[8];
    cd* acc[8];
    double c_next, b_acc;
    int first, last;
};
// R^ from the 16 transformed product fields and the state; mode 0: write R^ to rout only;
// mode 1: Euler update U += dt R, Rold = R; mode 2: AB2 update U += dt(1.5 R - 0.5 Rold), Rold = R; mode 3: `stage`
// force (or null): 4 arrays F^_x, F^_y, F^_z, (m.f)^ added to R_m and R_E (launch_forcing below)
void launch_assemble(const SpecGeom& g, const cd* const prod[16], cd* const U[8], cd* const Rold[8],
                     cd* const rout[8], int mode, double dt, Phys ph, cudaStream_t st, const cd* const force[4] = nullptr,
                     const cd* const visc[9] = nullptr, const StageUpdate* stage = nullptr);   // visc: V^xx,xy,xz,yy,yz,zz, Wv^x,y,z: R_m += i k_j V^_ij, R_E += i k.Wv^
// full stress tensor variant (Eq. 3-4, 11-12): u = m/rho in real space; S^ (xx,xy,xz,yy,yz,zz) from u^;
// V_ij = 2 nu rho S_ij (in place over S) and Wv_j = u_i V_ij in real space
void launch_velocity_real(long long n, const double* rho, const double* const m[3], double* const u[3], cudaStream_t st);
void launch_strain_spec(const SpecGeom& g, const cd* const u[3], cd* const S[6], Phys ph, cudaStream_t st);
void launch_viscous_flux(long long n, double nu, const double* rho, const double* const u[3], double* const SV[6],
                         double* const Wv[3], cudaStream_t st);
// ABC forcing in k-space (full layout only): F^ = M (rho f)^ and M (m.f)^ as +-kf shifts of rho^, m^ (exact: the
// state is band-limited to the mask).  add = 0: out[0..3] = F ; add = 1: out[1..4] += F (out = an 8-field R^ array)
void launch_forcing(const SpecGeom& g, const cd* const U[8], cd* const out[], int add, Phys ph, cudaStream_t st);
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
// slab-after-slab / brick-after-brick variants for the chunked pipeline: partials accumulate in a fixed order
void launch_diag_partial(long long n, const double* const U[8], double gamma, double* part, int accumulate, cudaStream_t st);
void launch_diag_final(const double* part, double* out, double inv_n, cudaStream_t st);
void launch_absmax_partial(long long n, const double* f, double* part, int accumulate, cudaStream_t st);
void launch_absmax_final(const double* part, double* out, cudaStream_t st);
void launch_shell_spectrum_compact(const SpecGeom& g, const cd* const spec[3], double* part, int nspec, int accumulate,
                                   cudaStream_t st);
void launch_shell_spectrum_final(const double* part, double* out, int nspec, cudaStream_t st);
int diag_partial_doubles();
int absmax_partial_doubles();
int spectrum_partial_doubles(int nspec);

// ---- tracer particles (tracers.cu) ------------------------------------------------------------------------
struct TracerArgs {
    const double* B[3];    // real-space grid fields [z][y][x] gathered by the push
    double* pos[3];
    double* vel[3];
    long long np;
    int N;
    double L, dt;
    int nsteps;            // pushes in the frozen field
};
void launch_tracer_push(const TracerArgs& a, cudaStream_t st);
// vel <- CIC interpolation of m/rho (real-space rho, mx, my, mz)
void launch_tracer_init_velocity(const TracerArgs& a, const double* rho, const double* const m[3], cudaStream_t st);
void launch_tracer_wrap(const TracerArgs& a, cudaStream_t st);
// spatial sort by grid row (see tracers.cu): (pos, vel, id) -> (alt[0..5], alt_id); hist holds N*N bins
void launch_tracer_sort(const TracerArgs& a, const long long* id, double* const alt[6], long long* alt_id, unsigned* hist,
                        unsigned* key, unsigned* rank, cudaStream_t st);
void launch_tracer_iota(long long np, long long* id, cudaStream_t st);
void launch_tracer_unpermute(long long np, const long long* id, const double* in, double* out, cudaStream_t st);

void launch_twiddle_table(int N, cd* tw, cudaStream_t st);

}  // namespace mhd

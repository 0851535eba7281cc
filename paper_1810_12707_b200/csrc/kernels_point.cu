// kernels_point.cu — point-wise kernels in k-space and real space, reductions for the diagnostics, twiddles.
//
// k-space kernels run over the half-spectrum arrays [kz][ky][kx] (row pitch hx = N/2 complex; the Nyquist
// column is not stored).  In pruned mode only the modes inside the 2/3 mask are visited — (2kc+1)^2 (kc+1) of
// N^2 N/2, i.e. 30 % — everything outside is identically zero by construction and is never read.
#include "fft_core.cuh"
#include "kernels.h"
#include "physics.cuh"

namespace mhd {

// ---- mode geometry -----------------------------------------------------------------------------------------
struct ModeIt {
    int ix, iy, iz;          // array indices (full layout) / compact indices (bricks)
    int nx, ny, nz;          // integer modes
    bool inside;             // inside the 2/3 mask
    long long idx;           // linear index into "work" arrays
    long long sidx;          // linear index into "state" arrays (same as idx in the full layout)
};
// grid: x over kx (blockDim.x threads), y over the (possibly pruned) ky count, z over the kz count
__device__ __forceinline__ bool mode_of_thread(const SpecGeom& g, ModeIt& m) {
    const int N = g.N, kc = g.kc;
    m.ix = blockIdx.x * blockDim.x + threadIdx.x;
    int oy = blockIdx.y, oz = blockIdx.z;
    if (g.compact) {
        if (m.ix > kc) return false;
        const int cy = oy + g.y0;
        m.iy = oy; m.iz = oz;
        m.nx = m.ix;
        m.ny = cy <= kc ? cy : cy - (2 * kc + 1);
        m.nz = oz <= kc ? oz : oz - (2 * kc + 1);
        m.inside = true;
        m.idx = (long long)oz * g.wsz + (long long)oy * g.wsy + m.ix;
        m.sidx = (long long)oz * g.ssz + (long long)oy * g.ssy + m.ix;
        return true;
    }
    if (g.pruned) {
        if (m.ix > kc) return false;
        m.iy = oy <= kc ? oy : N - (2 * kc + 1) + oy;
        m.iz = oz <= kc ? oz : N - (2 * kc + 1) + oz;
    } else {
        if (m.ix >= g.hx) return false;
        m.iy = oy; m.iz = oz;
    }
    m.nx = m.ix;
    m.ny = m.iy <= N / 2 ? m.iy : m.iy - N;
    m.nz = m.iz <= N / 2 ? m.iz : m.iz - N;
    m.inside = m.nx <= kc && abs(m.ny) <= kc && abs(m.nz) <= kc;
    m.idx = ((long long)m.iz * N + m.iy) * g.hx + m.ix;
    m.sidx = m.idx;
    return true;
}
static dim3 mode_grid(const SpecGeom& g, int threads) {
    if (g.compact) return dim3((g.kc + 1 + threads - 1) / threads, g.ny, 2 * g.kc + 1);
    const int nxv = g.pruned ? g.kc + 1 : g.hx;
    const int nyv = g.pruned ? 2 * g.kc + 1 : g.N;
    return dim3((nxv + threads - 1) / threads, nyv, nyv);
}
// threads along kx for the point-wise k-space kernels: 64, or 32 when that wastes fewer lanes on the last block of a row
// (N = 256: kc + 1 = 86 columns -> 3 x 32 instead of 2 x 64: 90 % instead of 67 % of the lanes carry a mode)
static int kt_for(const SpecGeom& g) {
    const int nxv = (g.compact || g.pruned) ? g.kc + 1 : g.hx;
    return ((nxv + 31) / 32) * 32 < ((nxv + 63) / 64) * 64 ? 32 : 64;
}

struct Ptr3 { const cd* p[3]; };
struct PtrW3 { cd* p[3]; };
struct Ptr8 { cd* p[8]; };
struct PtrC16 { const cd* p[16]; };
struct PtrN { cd* p[MAXF]; };
struct PtrCN { const cd* p[MAXF]; };

// ---- J^ = M i k x B^ -----------------------------------------------------------------------------------
__global__ void build_current_kernel(SpecGeom g, Ptr3 B, PtrW3 J, Phys ph) {
    ModeIt m;
    if (!mode_of_thread(g, m)) return;
    cd jx = mk(0, 0), jy = jx, jz = jx;
    if (m.inside) {
        const double kx = ph.k0 * m.nx, ky = ph.k0 * m.ny, kz = ph.k0 * m.nz;
        const cd bx = B.p[0][m.sidx], by = B.p[1][m.sidx], bz = B.p[2][m.sidx];
        jx = imul(ky, bz) - imul(kz, by);
        jy = imul(kz, bx) - imul(kx, bz);
        jz = imul(kx, by) - imul(ky, bx);
    }
    J.p[0][m.idx] = jx; J.p[1][m.idx] = jy; J.p[2][m.idx] = jz;
}
void launch_build_current(const SpecGeom& g, const cd* const B[3], cd* const J[3], Phys ph, cudaStream_t st) {
    Ptr3 b; PtrW3 j;
    for (int c = 0; c < 3; ++c) { b.p[c] = B[c]; j.p[c] = J[c]; }
    build_current_kernel<<<mode_grid(g, kt_for(g)), kt_for(g), 0, st>>>(g, b, j, ph);
}

// ---- div^ = M i k . B^ ---------------------------------------------------------------------------------
__global__ void divergence_kernel(SpecGeom g, Ptr3 B, cd* out, Phys ph) {
    ModeIt m;
    if (!mode_of_thread(g, m)) return;
    cd d = mk(0, 0);
    if (m.inside) {
        const double kx = ph.k0 * m.nx, ky = ph.k0 * m.ny, kz = ph.k0 * m.nz;
        d = imul(kx, B.p[0][m.sidx]) + imul(ky, B.p[1][m.sidx]) + imul(kz, B.p[2][m.sidx]);
    }
    out[m.idx] = d;
}
void launch_divergence(const SpecGeom& g, const cd* const B[3], cd* out, Phys ph, cudaStream_t st) {
    Ptr3 b;
    for (int c = 0; c < 3; ++c) b.p[c] = B[c];
    divergence_kernel<<<mode_grid(g, kt_for(g)), kt_for(g), 0, st>>>(g, b, out, ph);
}

// ---- R^ assembly (+ explicit update) -------------------------------------------------------------------
// mode 0: rout = R ; 1: U += dt R, Rold = R ; 2: U += dt (1.5 R - 0.5 Rold), Rold = R
struct PtrC4 { const cd* p[4]; };
struct PtrC9 { const cd* p[9]; };
// VAR = false: the default equation set (no forcing, no stress-tensor terms, nothing switched off) — the hot path keeps
// its register budget; VAR = true: all variants of DESIGN.md section 13
template <bool VAR>
__global__ void assemble_kernel(SpecGeom g, PtrC16 pr, Ptr8 U, Ptr8 Rold, Ptr8 rout, int mode, double dt, Phys ph, PtrC4 force,
                                PtrC9 visc, StageUpdate sg) {
    ModeIt m;
    if (!mode_of_thread(g, m)) return;
    const long long i = m.idx, j = m.sidx;     // products / state
    cd R[8];
    if (m.inside) {
        const double kx = ph.k0 * m.nx, ky = ph.k0 * m.ny, kz = ph.k0 * m.nz;
        cd u[8];
#pragma unroll
        for (int f = 0; f < 8; ++f) u[f] = U.p[f][j];
        rhs_mode([&](int s) { return pr.p[s][i]; }, u, kx, ky, kz, ph, R);
        if constexpr (VAR) {
        if (visc.p[0]) {         // variant: + d_j (2 nu rho S_ij) and + d_j (2 nu rho u_i S_ij)  (Eq. 11-12)
            const cd vxx = visc.p[0][j], vxy = visc.p[1][j], vxz = visc.p[2][j], vyy = visc.p[3][j], vyz = visc.p[4][j], vzz = visc.p[5][j];
            R[1] = R[1] + (imul(kx, vxx) + imul(ky, vxy) + imul(kz, vxz));
            R[2] = R[2] + (imul(kx, vxy) + imul(ky, vyy) + imul(kz, vyz));
            R[3] = R[3] + (imul(kx, vxz) + imul(ky, vyz) + imul(kz, vzz));
            R[4] = R[4] + (imul(kx, visc.p[6][j]) + imul(ky, visc.p[7][j]) + imul(kz, visc.p[8][j]));
        }
        if (force.p[0]) {        // variants: rho f and its work m.f (launch_forcing), state geometry
#pragma unroll
            for (int f = 0; f < 4; ++f) R[1 + f] = R[1 + f] + force.p[f][j];
        }
        if (ph.cs2 > 0.0) R[4] = mk(0, 0);                      // barotropic: no energy equation
        if (!(ph.evolve & 1)) { R[0] = R[1] = R[2] = R[3] = R[4] = mk(0, 0); }
        if (!(ph.evolve & 2)) { R[5] = R[6] = R[7] = mk(0, 0); }
        }
        if (mode == 0) {
#pragma unroll
            for (int f = 0; f < 8; ++f) rout.p[f][i] = R[f];     // work-array geometry (may alias the products)
        } else if (mode == 3) {      // one stage of RK4 / predictor-corrector, low-storage form (kernels.h StageUpdate)
#pragma unroll
            for (int f = 0; f < 8; ++f) {
                const cd u0 = sg.first ? u[f] : sg.U0[f][j];
                const cd a = sg.first ? mk(0, 0) : sg.acc[f][j];
                if (sg.first) sg.U0[f][j] = u[f];
                const cd an = mk(a.x + sg.b_acc * R[f].x, a.y + sg.b_acc * R[f].y);
                if (sg.last) U.p[f][j] = mk(u0.x + an.x, u0.y + an.y);
                else {
                    sg.acc[f][j] = an;
                    U.p[f][j] = mk(u0.x + sg.c_next * R[f].x, u0.y + sg.c_next * R[f].y);
                }
            }
        } else {
#pragma unroll
            for (int f = 0; f < 8; ++f) {
                const cd ro = mode == 2 ? Rold.p[f][j] : mk(0, 0);
                U.p[f][j] = updated(mode, dt, u[f], R[f], ro);
                Rold.p[f][j] = R[f];
            }
        }
    } else if (mode == 0) {      // unpruned sweep: make the masked-out modes explicit zeros
#pragma unroll
        for (int f = 0; f < 8; ++f) rout.p[f][i] = mk(0, 0);
    }
}
void launch_assemble(const SpecGeom& g, const cd* const prod[16], cd* const U[8], cd* const Rold[8],
                     cd* const rout[8], int mode, double dt, Phys ph, cudaStream_t st, const cd* const force[4],
                     const cd* const visc[9], const StageUpdate* stage) {
    PtrC16 p; Ptr8 u, ro, rr; PtrC4 fc; PtrC9 vc;
    for (int f = 0; f < 9; ++f) vc.p[f] = visc ? visc[f] : nullptr;
    for (int f = 0; f < 4; ++f) fc.p[f] = force ? force[f] : nullptr;
    for (int f = 0; f < 16; ++f) p.p[f] = prod[f];
    for (int f = 0; f < 8; ++f) { u.p[f] = U[f]; ro.p[f] = Rold ? Rold[f] : nullptr; rr.p[f] = rout ? rout[f] : nullptr; }
    const bool var = force || visc || ph.cs2 > 0.0 || ph.evolve != 3;
    StageUpdate sg = StageUpdate();
    if (stage) sg = *stage;
    if (var) assemble_kernel<true><<<mode_grid(g, kt_for(g)), kt_for(g), 0, st>>>(g, p, u, ro, rr, mode, dt, ph, fc, vc, sg);
    else assemble_kernel<false><<<mode_grid(g, kt_for(g)), kt_for(g), 0, st>>>(g, p, u, ro, rr, mode, dt, ph, fc, vc, sg);
}

// ---- full stress tensor variant (Eq. 3-4, 11-12) -------------------------------------------------------
struct PtrW6 { cd* p[6]; };
// S^_ij = i (k_i u^_j + k_j u^_i)/2 - delta_ij i k.u^/3 on the masked modes; slot order xx, xy, xz, yy, yz, zz
__global__ void strain_spec_kernel(SpecGeom g, Ptr3 u, PtrW6 S, Phys ph) {
    ModeIt m;
    if (!mode_of_thread(g, m) || !m.inside) return;
    const double kx = ph.k0 * m.nx, ky = ph.k0 * m.ny, kz = ph.k0 * m.nz;
    const cd ux = u.p[0][m.idx], uy = u.p[1][m.idx], uz = u.p[2][m.idx];
    const cd dxx = imul(kx, ux), dyy = imul(ky, uy), dzz = imul(kz, uz);
    const cd th3 = (1.0 / 3.0) * (dxx + dyy + dzz);
    S.p[0][m.idx] = dxx - th3;
    S.p[1][m.idx] = 0.5 * (imul(kx, uy) + imul(ky, ux));
    S.p[2][m.idx] = 0.5 * (imul(kx, uz) + imul(kz, ux));
    S.p[3][m.idx] = dyy - th3;
    S.p[4][m.idx] = 0.5 * (imul(ky, uz) + imul(kz, uy));
    S.p[5][m.idx] = dzz - th3;
}
void launch_strain_spec(const SpecGeom& g, const cd* const u[3], cd* const S[6], Phys ph, cudaStream_t st) {
    Ptr3 uu; PtrW6 ss;
    for (int c = 0; c < 3; ++c) uu.p[c] = u[c];
    for (int c = 0; c < 6; ++c) ss.p[c] = S[c];
    strain_spec_kernel<<<mode_grid(g, kt_for(g)), kt_for(g), 0, st>>>(g, uu, ss, ph);
}

// ---- ABC forcing in k-space ------------------------------------------------------------------------------
// a^(n) of a real field from its half spectrum (nx >= 0 stored; Hermitian symmetry for nx < 0); zero outside the mask
__device__ __forceinline__ cd spec_at(const cd* __restrict__ a, int N, int hx, int kc, int nx, int ny, int nz) {
    if (abs(nx) > kc || abs(ny) > kc || abs(nz) > kc) return mk(0, 0);
    const bool neg = nx < 0;
    if (neg) { nx = -nx; ny = -ny; nz = -nz; }
    const int iy = ny >= 0 ? ny : ny + N, iz = nz >= 0 ? nz : nz + N;
    const cd v = a[((long long)iz * N + iy) * hx + nx];
    return neg ? cconj(v) : v;
}
// (a sin(kf x_d))^(n) = (a^(n - kf e_d) - a^(n + kf e_d)) / (2i) ;  (a cos(kf x_d))^(n) = (a^(n - kf e_d) + a^(n + kf e_d)) / 2
__device__ __forceinline__ void shifted(const cd* __restrict__ a, const SpecGeom& g, const ModeIt& m, int d, int kf, cd& lo, cd& hi) {
    const int dx = d == 0 ? kf : 0, dy = d == 1 ? kf : 0, dz = d == 2 ? kf : 0;
    lo = spec_at(a, g.N, g.hx, g.kc, m.nx - dx, m.ny - dy, m.nz - dz);
    hi = spec_at(a, g.N, g.hx, g.kc, m.nx + dx, m.ny + dy, m.nz + dz);
}
__device__ __forceinline__ cd times_sin(const cd* a, const SpecGeom& g, const ModeIt& m, int d, int kf) {
    cd lo, hi; shifted(a, g, m, d, kf, lo, hi);
    const cd df = lo - hi;
    return mk(0.5 * df.y, -0.5 * df.x);      // / (2i)
}
__device__ __forceinline__ cd times_cos(const cd* a, const SpecGeom& g, const ModeIt& m, int d, int kf) {
    cd lo, hi; shifted(a, g, m, d, kf, lo, hi);
    return 0.5 * (lo + hi);
}
__global__ void forcing_kernel(SpecGeom g, Ptr8 U, Ptr8 out, int add, Phys ph) {
    ModeIt m;
    if (!mode_of_thread(g, m) || !m.inside) return;
    const int kf = ph.kf;
    // f = f0 (sin kz + cos ky, sin kx + cos kz, sin ky + cos kx)    (A = B = C = 1)
    cd F[4];
    F[0] = ph.f0 * (times_sin(U.p[0], g, m, 2, kf) + times_cos(U.p[0], g, m, 1, kf));
    F[1] = ph.f0 * (times_sin(U.p[0], g, m, 0, kf) + times_cos(U.p[0], g, m, 2, kf));
    F[2] = ph.f0 * (times_sin(U.p[0], g, m, 1, kf) + times_cos(U.p[0], g, m, 0, kf));
    F[3] = ph.f0 * (times_sin(U.p[1], g, m, 2, kf) + times_cos(U.p[1], g, m, 1, kf)
                    + times_sin(U.p[2], g, m, 0, kf) + times_cos(U.p[2], g, m, 2, kf)
                    + times_sin(U.p[3], g, m, 1, kf) + times_cos(U.p[3], g, m, 0, kf));
    if (ph.cs2 > 0.0) F[3] = mk(0, 0);
    if (!(ph.evolve & 1)) F[0] = F[1] = F[2] = F[3] = mk(0, 0);
#pragma unroll
    for (int f = 0; f < 4; ++f) {
        if (add) out.p[1 + f][m.idx] = out.p[1 + f][m.idx] + F[f];
        else out.p[f][m.idx] = F[f];
    }
}
void launch_forcing(const SpecGeom& g, const cd* const U[8], cd* const out[], int add, Phys ph, cudaStream_t st) {
    Ptr8 u, o;
    for (int f = 0; f < 8; ++f) { u.p[f] = const_cast<cd*>(U[f]); o.p[f] = nullptr; }
    for (int f = 0; f < (add ? 8 : 4); ++f) o.p[f] = out[f];
    forcing_kernel<<<mode_grid(g, kt_for(g)), kt_for(g), 0, st>>>(g, u, o, add, ph);
}

// ---- y = a y + b x on the masked modes (integrator stages) -----------------------------------------------
__global__ void axpby_kernel(SpecGeom g, int nf, double a, PtrN y, double b, PtrCN x) {
    ModeIt m;
    if (!mode_of_thread(g, m) || !m.inside) return;
    for (int f = 0; f < nf; ++f) {
        const cd xv = x.p[f][m.idx];
        cd yv = mk(0, 0);
        if (a != 0.0) { yv = y.p[f][m.sidx]; yv = mk(a * yv.x, a * yv.y); }
        y.p[f][m.sidx] = mk(yv.x + b * xv.x, yv.y + b * xv.y);
    }
}
void launch_axpby(const SpecGeom& g, int nf, double a, cd* const y[], double b, const cd* const x[], cudaStream_t st) {
    PtrN yy; PtrCN xx;
    for (int f = 0; f < nf; ++f) { yy.p[f] = y[f]; xx.p[f] = x[f]; }
    axpby_kernel<<<mode_grid(g, kt_for(g)), kt_for(g), 0, st>>>(g, nf, a, yy, b, xx);
}
void launch_copy_masked(const SpecGeom& g, int nf, cd* const dst[], const cd* const src[], cudaStream_t st) {
    launch_axpby(g, nf, 0.0, dst, 1.0, src, st);
}

// ---- zero the modes outside the mask (unpruned sweep over everything stored) -----------------------------
__global__ void zero_outside_kernel(SpecGeom g, int nf, PtrN f) {
    ModeIt m;
    if (!mode_of_thread(g, m) || m.inside) return;
    for (int c = 0; c < nf; ++c) f.p[c][m.idx] = mk(0, 0);
}
void launch_zero_outside_mask(const SpecGeom& g0, int nf, cd* const f[], cudaStream_t st) {
    SpecGeom g = g0; g.pruned = 0;
    PtrN p;
    for (int c = 0; c < nf; ++c) p.p[c] = f[c];
    zero_outside_kernel<<<mode_grid(g, kt_for(g)), kt_for(g), 0, st>>>(g, nf, p);
}

// ---- real-space point-wise kernels -----------------------------------------------------------------------
struct PtrR11 { const double* p[11]; };
struct PtrR16 { double* p[16]; };
struct PtrR8 { double* p[8]; };
struct PtrRC8 { const double* p[8]; };
struct PtrRW3 { double* p[3]; };

__global__ void flux_real_kernel(long long n, PtrR11 in, PtrR16 out, Phys ph) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        double s[S_NIN], o[P_NOUT];
#pragma unroll
        for (int f = 0; f < S_NIN; ++f) s[f] = in.p[f][i];
        flux_point(s, o, ph);
#pragma unroll
        for (int f = 0; f < P_NOUT; ++f) out.p[f][i] = o[f];
    }
}
static int ew_blocks(long long n, int threads) {
    long long b = (n + threads - 1) / threads;
    const long long cap = 148LL * 16;
    return (int)(b < cap ? b : cap);
}
void launch_flux_real(long long n, const double* const in[11], double* const out[16], Phys ph, cudaStream_t st) {
    PtrR11 a; PtrR16 b;
    for (int f = 0; f < 11; ++f) a.p[f] = in[f];
    for (int f = 0; f < 16; ++f) b.p[f] = out[f];
    flux_real_kernel<<<ew_blocks(n, 256), 256, 0, st>>>(n, a, b, ph);
}

struct PtrRC3 { const double* p[3]; };
struct PtrRW6 { double* p[6]; };
__global__ void velocity_real_kernel(long long n, const double* rho, PtrRC3 m, PtrRW3 u) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const double r = rho[i];
        u.p[0][i] = m.p[0][i] / r; u.p[1][i] = m.p[1][i] / r; u.p[2][i] = m.p[2][i] / r;
    }
}
void launch_velocity_real(long long n, const double* rho, const double* const m[3], double* const u[3], cudaStream_t st) {
    PtrRC3 mm; PtrRW3 uu;
    for (int c = 0; c < 3; ++c) { mm.p[c] = m[c]; uu.p[c] = u[c]; }
    velocity_real_kernel<<<ew_blocks(n, 256), 256, 0, st>>>(n, rho, mm, uu);
}
// V_ij = 2 nu rho S_ij in place; Wv_j = u_i V_ij
__global__ void viscous_flux_kernel(long long n, double nu, const double* rho, PtrRC3 u, PtrRW6 SV, PtrRW3 Wv) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const double f = 2.0 * nu * rho[i];
        const double vxx = f * SV.p[0][i], vxy = f * SV.p[1][i], vxz = f * SV.p[2][i];
        const double vyy = f * SV.p[3][i], vyz = f * SV.p[4][i], vzz = f * SV.p[5][i];
        const double ux = u.p[0][i], uy = u.p[1][i], uz = u.p[2][i];
        SV.p[0][i] = vxx; SV.p[1][i] = vxy; SV.p[2][i] = vxz; SV.p[3][i] = vyy; SV.p[4][i] = vyz; SV.p[5][i] = vzz;
        Wv.p[0][i] = ux * vxx + uy * vxy + uz * vxz;
        Wv.p[1][i] = ux * vxy + uy * vyy + uz * vyz;
        Wv.p[2][i] = ux * vxz + uy * vyz + uz * vzz;
    }
}
void launch_viscous_flux(long long n, double nu, const double* rho, const double* const u[3], double* const SV[6],
                         double* const Wv[3], cudaStream_t st) {
    PtrRC3 uu; PtrRW6 ss; PtrRW3 ww;
    for (int c = 0; c < 3; ++c) { uu.p[c] = u[c]; ww.p[c] = Wv[c]; }
    for (int c = 0; c < 6; ++c) ss.p[c] = SV[c];
    viscous_flux_kernel<<<ew_blocks(n, 256), 256, 0, st>>>(n, nu, rho, uu, ss, ww);
}

__global__ void prim_to_cons_kernel(long long n, PtrR8 f, double gamma) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const double rho = f.p[0][i], ux = f.p[1][i], uy = f.p[2][i], uz = f.p[3][i], P = f.p[4][i];
        const double bx = f.p[5][i], by = f.p[6][i], bz = f.p[7][i];
        f.p[1][i] = rho * ux; f.p[2][i] = rho * uy; f.p[3][i] = rho * uz;
        f.p[4][i] = P / (gamma - 1.0) + 0.5 * rho * (ux * ux + uy * uy + uz * uz) + 0.5 * (bx * bx + by * by + bz * bz);
    }
}
void launch_prim_to_cons(long long n, double* const f[8], double gamma, cudaStream_t st) {
    PtrR8 a;
    for (int c = 0; c < 8; ++c) a.p[c] = f[c];
    prim_to_cons_kernel<<<ew_blocks(n, 256), 256, 0, st>>>(n, a, gamma);
}
__global__ void cons_to_prim_kernel(long long n, PtrR8 f, double gamma) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const double rho = f.p[0][i], mx = f.p[1][i], my = f.p[2][i], mz = f.p[3][i], E = f.p[4][i];
        const double bx = f.p[5][i], by = f.p[6][i], bz = f.p[7][i];
        const double ux = mx / rho, uy = my / rho, uz = mz / rho;
        f.p[1][i] = ux; f.p[2][i] = uy; f.p[3][i] = uz;
        f.p[4][i] = (gamma - 1.0) * (E - 0.5 * (mx * ux + my * uy + mz * uz) - 0.5 * (bx * bx + by * by + bz * bz));
    }
}
void launch_cons_to_prim(long long n, double* const f[8], double gamma, cudaStream_t st) {
    PtrR8 a;
    for (int c = 0; c < 8; ++c) a.p[c] = f[c];
    cons_to_prim_kernel<<<ew_blocks(n, 256), 256, 0, st>>>(n, a, gamma);
}

__global__ void sqrt_rho_u_kernel(long long n, PtrRC8 U, PtrRW3 w) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const double s = 1.0 / sqrt(U.p[0][i]);
        w.p[0][i] = U.p[1][i] * s; w.p[1][i] = U.p[2][i] * s; w.p[2][i] = U.p[3][i] * s;
    }
}
void launch_sqrt_rho_u(long long n, const double* const U[8], double* const w[3], cudaStream_t st) {
    PtrRC8 a; PtrRW3 b;
    for (int c = 0; c < 8; ++c) a.p[c] = U[c];
    for (int c = 0; c < 3; ++c) b.p[c] = w[c];
    sqrt_rho_u_kernel<<<ew_blocks(n, 256), 256, 0, st>>>(n, a, b);
}

// ---- reductions: fixed grid, fixed tree order -> bitwise reproducible (the scalar diagnostics; the shell spectra below
//      bin with shared-memory atomicAdd inside a block: reproducible to roundoff only) ---------------------------------
constexpr int RB = 1024;     // blocks of the first stage
constexpr int RT = 256;      // threads per block
constexpr int NRED = 10;     // ke, me, ie, mass, momx, momy, momz, etot (sums); rho_min, p_min

__device__ __forceinline__ void block_reduce(double (&v)[NRED], double* sh /*[NRED][RT]*/) {
    const int t = threadIdx.x;
#pragma unroll
    for (int q = 0; q < NRED; ++q) sh[q * RT + t] = v[q];
    __syncthreads();
    for (int s = RT / 2; s > 0; s >>= 1) {
        if (t < s) {
#pragma unroll
            for (int q = 0; q < NRED; ++q) {
                const double a = sh[q * RT + t], b = sh[q * RT + t + s];
                sh[q * RT + t] = (q < 8) ? a + b : fmin(a, b);
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int q = 0; q < NRED; ++q) v[q] = sh[q * RT];
}

__global__ void __launch_bounds__(RT) diag_stage1(long long n, PtrRC8 U, double gamma, double* part /*[RB][NRED]*/, int accumulate) {
    __shared__ double sh[NRED * RT];
    double v[NRED];
#pragma unroll
    for (int q = 0; q < 8; ++q) v[q] = 0.0;
    v[8] = v[9] = 1e300;
    for (long long i = blockIdx.x * (long long)RT + threadIdx.x; i < n; i += (long long)RB * RT) {
        const double rho = U.p[0][i], mx = U.p[1][i], my = U.p[2][i], mz = U.p[3][i], E = U.p[4][i];
        const double bx = U.p[5][i], by = U.p[6][i], bz = U.p[7][i];
        const double ux = mx / rho, uy = my / rho, uz = mz / rho;
        const double k = 0.5 * (mx * ux + my * uy + mz * uz), hb = 0.5 * (bx * bx + by * by + bz * bz);
        const double P = (gamma - 1.0) * (E - k - hb);
        v[0] += k; v[1] += hb; v[2] += P / (gamma - 1.0); v[3] += rho; v[4] += mx; v[5] += my; v[6] += mz; v[7] += E;
        v[8] = fmin(v[8], rho); v[9] = fmin(v[9], P);
    }
    block_reduce(v, sh);
    if (threadIdx.x == 0)
        for (int q = 0; q < NRED; ++q) {
            double* p = &part[blockIdx.x * NRED + q];
            *p = !accumulate ? v[q] : (q < 8 ? *p + v[q] : fmin(*p, v[q]));     // slab after slab, fixed order
        }
}
__global__ void __launch_bounds__(RT) diag_stage2(const double* part, double* out, double inv_n) {
    __shared__ double sh[NRED * RT];
    double v[NRED];
#pragma unroll
    for (int q = 0; q < 8; ++q) v[q] = 0.0;
    v[8] = v[9] = 1e300;
    for (int b = threadIdx.x; b < RB; b += RT)
        for (int q = 0; q < NRED; ++q) {
            const double x = part[b * NRED + q];
            v[q] = (q < 8) ? v[q] + x : fmin(v[q], x);
        }
    block_reduce(v, sh);
    if (threadIdx.x == 0)
        for (int q = 0; q < NRED; ++q) out[q] = (q < 8) ? v[q] * inv_n : v[q];
}
void launch_diag_reduce(long long n, const double* const U[8], double gamma, double* scratch, double* out,
                        cudaStream_t st) {
    PtrRC8 a;
    for (int c = 0; c < 8; ++c) a.p[c] = U[c];
    diag_stage1<<<RB, RT, 0, st>>>(n, a, gamma, scratch, 0);
    diag_stage2<<<1, RT, 0, st>>>(scratch, out, 1.0 / (double)n);
}
void launch_diag_partial(long long n, const double* const U[8], double gamma, double* part, int accumulate, cudaStream_t st) {
    PtrRC8 a;
    for (int c = 0; c < 8; ++c) a.p[c] = U[c];
    diag_stage1<<<RB, RT, 0, st>>>(n, a, gamma, part, accumulate);
}
void launch_diag_final(const double* part, double* out, double inv_n, cudaStream_t st) {
    diag_stage2<<<1, RT, 0, st>>>(part, out, inv_n);
}
int diag_partial_doubles() { return RB * NRED; }
int absmax_partial_doubles() { return RB; }

__global__ void __launch_bounds__(RT) absmax_stage1(long long n, const double* f, double* part, int accumulate) {
    __shared__ double sh[RT];
    double v = 0.0;
    for (long long i = blockIdx.x * (long long)RT + threadIdx.x; i < n; i += (long long)RB * RT) v = fmax(v, fabs(f[i]));
    sh[threadIdx.x] = v;
    __syncthreads();
    for (int s = RT / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] = fmax(sh[threadIdx.x], sh[threadIdx.x + s]);
        __syncthreads();
    }
    if (threadIdx.x == 0) part[blockIdx.x] = accumulate ? fmax(part[blockIdx.x], sh[0]) : sh[0];
}
__global__ void __launch_bounds__(RT) absmax_stage2(const double* part, double* out) {
    __shared__ double sh[RT];
    double v = 0.0;
    for (int b = threadIdx.x; b < RB; b += RT) v = fmax(v, part[b]);
    sh[threadIdx.x] = v;
    __syncthreads();
    for (int s = RT / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] = fmax(sh[threadIdx.x], sh[threadIdx.x + s]);
        __syncthreads();
    }
    if (threadIdx.x == 0) out[0] = sh[0];
}
void launch_absmax(long long n, const double* f, double* scratch, double* out, cudaStream_t st) {
    absmax_stage1<<<RB, RT, 0, st>>>(n, f, scratch, 0);
    absmax_stage2<<<1, RT, 0, st>>>(scratch, out);
}
void launch_absmax_partial(long long n, const double* f, double* part, int accumulate, cudaStream_t st) {
    absmax_stage1<<<RB, RT, 0, st>>>(n, f, part, accumulate);
}
void launch_absmax_final(const double* part, double* out, cudaStream_t st) { absmax_stage2<<<1, RT, 0, st>>>(part, out); }

// ---- shell spectra ---------------------------------------------------------------------------------------
// S(K) = sum over the FULL mode cube with floor(|n|+1/2) = K of 1/2 sum_c |w^_c(n)|^2 / N^6.  The stored half
// spectrum counts kx = 1..N/2-1 twice (the conjugate half), kx = 0 and the Nyquist plane once.
constexpr int SB = 512;      // blocks of the first stage
constexpr int MAXSPEC = 1024;
int diag_scratch_doubles(int nspec) { int a = SB * nspec, b = RB * NRED; return a > b ? a : b; }

__global__ void __launch_bounds__(256) spectrum_stage1(int N, Ptr3 spec, Ptr3 nyq, double* part /*[SB][nspec]*/, int nspec) {
    __shared__ double hist[MAXSPEC];
    for (int k = threadIdx.x; k < nspec; k += blockDim.x) hist[k] = 0.0;
    __syncthreads();
    const int hx = N / 2;
    const long long nmain = (long long)N * N * hx, nny = (long long)N * N;
    const double n3 = (double)N * N * N, norm = 0.5 / (n3 * n3);
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < nmain + nny; i += (long long)SB * blockDim.x) {
        int ix, iy, iz; double e = 0.0, wgt;
        if (i < nmain) {
            ix = (int)(i % hx); iy = (int)((i / hx) % N); iz = (int)(i / ((long long)hx * N));
            for (int c = 0; c < 3; ++c) { const cd a = spec.p[c][i]; e += a.x * a.x + a.y * a.y; }
            wgt = ix == 0 ? 1.0 : 2.0;
        } else {
            const long long r = i - nmain;
            ix = hx; iy = (int)(r % N); iz = (int)(r / N);
            if (nyq.p[0]) for (int c = 0; c < 3; ++c) { const cd a = nyq.p[c][r * 8]; e += a.x * a.x + a.y * a.y; }
            wgt = 1.0;
        }
        const int ny = iy <= N / 2 ? iy : iy - N, nz = iz <= N / 2 ? iz : iz - N;
        const int K = (int)floor(sqrt((double)(ix * ix + ny * ny + nz * nz)) + 0.5);
        if (e != 0.0) atomicAdd(&hist[K], wgt * norm * e);
    }
    __syncthreads();
    for (int k = threadIdx.x; k < nspec; k += blockDim.x) part[(long long)blockIdx.x * nspec + k] = hist[k];
}
__global__ void spectrum_stage2(const double* part, double* out, int nspec) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nspec) return;
    double s = 0.0;
    for (int b = 0; b < SB; ++b) s += part[(long long)b * nspec + k];
    out[k] = s;
}
// compact bricks (chunked pipeline): only modes inside the mask are stored; partial sums accumulate brick after brick
__global__ void __launch_bounds__(256) spectrum_compact_stage1(SpecGeom g, Ptr3 spec, double* part, int nspec, int accumulate) {
    __shared__ double hist[MAXSPEC];
    for (int k = threadIdx.x; k < nspec; k += blockDim.x) hist[k] = 0.0;
    __syncthreads();
    const int kc = g.kc, nxv = kc + 1, nzc = 2 * kc + 1;
    const long long total = (long long)nxv * g.ny * nzc;
    const double n3 = (double)g.N * g.N * g.N, norm = 0.5 / (n3 * n3);
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)SB * blockDim.x) {
        const int ix = (int)(i % nxv), oy = (int)((i / nxv) % g.ny), oz = (int)(i / ((long long)nxv * g.ny));
        const int cy = oy + g.y0;
        const int ny = cy <= kc ? cy : cy - nzc, nz = oz <= kc ? oz : oz - nzc;
        const long long j = (long long)oz * g.ssz + (long long)oy * g.ssy + ix;
        double e = 0.0;
        for (int c = 0; c < 3; ++c) { const cd a = spec.p[c][j]; e += a.x * a.x + a.y * a.y; }
        const int K = (int)floor(sqrt((double)(ix * ix + ny * ny + nz * nz)) + 0.5);
        if (e != 0.0) atomicAdd(&hist[K], (ix == 0 ? 1.0 : 2.0) * norm * e);
    }
    __syncthreads();
    for (int k = threadIdx.x; k < nspec; k += blockDim.x) {
        double* p = &part[(long long)blockIdx.x * nspec + k];
        *p = accumulate ? *p + hist[k] : hist[k];
    }
}
void launch_shell_spectrum_compact(const SpecGeom& g, const cd* const spec[3], double* part, int nspec, int accumulate,
                                   cudaStream_t st) {
    Ptr3 a;
    for (int c = 0; c < 3; ++c) a.p[c] = spec[c];
    spectrum_compact_stage1<<<SB, 256, 0, st>>>(g, a, part, nspec, accumulate);
}
void launch_shell_spectrum_final(const double* part, double* out, int nspec, cudaStream_t st) {
    spectrum_stage2<<<(nspec + 127) / 128, 128, 0, st>>>(part, out, nspec);
}
int spectrum_partial_doubles(int nspec) { return SB * nspec; }

void launch_shell_spectrum(int N, const cd* const spec[3], const cd* const nyq[3], double* scratch, double* out,
                           int nspec, cudaStream_t st) {
    Ptr3 a, b;
    for (int c = 0; c < 3; ++c) { a.p[c] = spec[c]; b.p[c] = nyq ? nyq[c] : nullptr; }
    spectrum_stage1<<<SB, 256, 0, st>>>(N, a, b, scratch, nspec);
    spectrum_stage2<<<(nspec + 127) / 128, 128, 0, st>>>(scratch, out, nspec);
}

// ---- twiddle table: w[m] = exp(-2 pi i m / N), exactly rounded sincospi, no recurrences -------------------
__global__ void twiddle_kernel(int N, cd* tw) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= N) return;
    double s, c;
    sincospi(2.0 * (double)m / (double)N, &s, &c);
    tw[m] = mk(c, -s);
}
void launch_twiddle_table(int N, cd* tw, cudaStream_t st) { twiddle_kernel<<<(N + 127) / 128, 128, 0, st>>>(N, tw); }

}  // namespace mhd

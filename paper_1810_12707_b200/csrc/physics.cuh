// physics.cuh — point-wise arithmetic of the MHD right-hand side (device inline functions).
//
// Real space (Eq. 17-19, Eq. 12 L96 in normalised units; readings R1-R4):
//   u = m/rho,  P = (gamma-1)(E - m.u/2 - |B|^2/2),  Pt = P + |B|^2/2
//   T_ij  = m_i u_j + Pt delta_ij - B_i B_j                      (momentum flux, symmetric, 6 components)
//   F_E   = (E + Pt) u - (u.B) B - eta B x J                     (energy flux; J = curl B)
//   eps   = u x B                                                (dB/dt = curl eps + eta lap B)
//   u, q = |u|^2/2                                               (for mu lap u and mu lap q)
// Spectral space (derivative = multiplication by i k; mask applied by the caller):
//   R_rho = -i k.m^ ;  R_mi = -i k_j T^_ij - mu k^2 u^_i ;  R_E = -i k.F^_E - mu k^2 q^ ;
//   R_B   = i k x eps^ - eta k^2 B^
#pragma once
#include "fft_core.cuh"
#include "kernels.h"

namespace mhd {

// slot order of the 11 real-space inputs and 16 products
enum { S_RHO = 0, S_MX, S_MY, S_MZ, S_E, S_BX, S_BY, S_BZ, S_JX, S_JY, S_JZ, S_NIN };
enum { P_TXX = 0, P_TXY, P_TXZ, P_TYY, P_TYZ, P_TZZ, P_FEX, P_FEY, P_FEZ, P_EX, P_EY, P_EZ, P_UX, P_UY, P_UZ, P_Q, P_NOUT };

__device__ __forceinline__ void flux_point(const double (&s)[S_NIN], double (&o)[P_NOUT], const Phys& ph) {
    const double ir = 1.0 / s[S_RHO];
    const double ux = s[S_MX] * ir, uy = s[S_MY] * ir, uz = s[S_MZ] * ir;
    const double bx = s[S_BX], by = s[S_BY], bz = s[S_BZ];
    const double b2 = bx * bx + by * by + bz * bz;
    const double mu_dot = s[S_MX] * ux + s[S_MY] * uy + s[S_MZ] * uz;
    const double P = ph.cs2 > 0.0 ? ph.cs2 * s[S_RHO]                                   // barotropic closure (Eq. 5 / 18)
                                  : (ph.gamma - 1.0) * (s[S_E] - 0.5 * mu_dot - 0.5 * b2);
    const double Pt = P + 0.5 * b2;
    o[P_TXX] = s[S_MX] * ux + Pt - bx * bx;
    o[P_TXY] = s[S_MX] * uy - bx * by;
    o[P_TXZ] = s[S_MX] * uz - bx * bz;
    o[P_TYY] = s[S_MY] * uy + Pt - by * by;
    o[P_TYZ] = s[S_MY] * uz - by * bz;
    o[P_TZZ] = s[S_MZ] * uz + Pt - bz * bz;
    const double udb = ux * bx + uy * by + uz * bz;
    const double h = s[S_E] + Pt;
    const double jx = s[S_JX], jy = s[S_JY], jz = s[S_JZ];
    o[P_FEX] = h * ux - udb * bx - ph.eta * (by * jz - bz * jy);
    o[P_FEY] = h * uy - udb * by - ph.eta * (bz * jx - bx * jz);
    o[P_FEZ] = h * uz - udb * bz - ph.eta * (bx * jy - by * jx);
    o[P_EX] = uy * bz - uz * by;
    o[P_EY] = uz * bx - ux * bz;
    o[P_EZ] = ux * by - uy * bx;
    o[P_UX] = ux; o[P_UY] = uy; o[P_UZ] = uz;
    o[P_Q] = 0.5 * (ux * ux + uy * uy + uz * uz);
}

// i * k * a  for real k
__device__ __forceinline__ cd imul(double k, cd a) { return mk(-k * a.y, k * a.x); }

// R^ of one mode (default equation set) from the 16 transformed products, fetched through ld(slot), and the state u[8]:
// derivative = multiplication by i k (PAPER.md L17 / L25), diffusion = -k^2 (Eq. 18-19).  One definition for
// assemble_kernel and for the assembly tail of the fused forward z pass, so that both give bitwise the same numbers.
template <class LD>
__device__ __forceinline__ void rhs_mode(LD ld, const cd (&u)[8], double kx, double ky, double kz, const Phys& ph, cd (&R)[8]) {
    const double k2 = kx * kx + ky * ky + kz * kz;
    const cd txx = ld(P_TXX), txy = ld(P_TXY), txz = ld(P_TXZ);
    const cd tyy = ld(P_TYY), tyz = ld(P_TYZ), tzz = ld(P_TZZ);
    const cd ex = ld(P_EX), ey = ld(P_EY), ez = ld(P_EZ);
    // -i k.F = -(i kx Fx + i ky Fy + i kz Fz)
    R[0] = mk(0, 0) - (imul(kx, u[1]) + imul(ky, u[2]) + imul(kz, u[3]));
    R[1] = mk(0, 0) - (imul(kx, txx) + imul(ky, txy) + imul(kz, txz)) - (ph.mu * k2) * ld(P_UX);
    R[2] = mk(0, 0) - (imul(kx, txy) + imul(ky, tyy) + imul(kz, tyz)) - (ph.mu * k2) * ld(P_UY);
    R[3] = mk(0, 0) - (imul(kx, txz) + imul(ky, tyz) + imul(kz, tzz)) - (ph.mu * k2) * ld(P_UZ);
    R[4] = mk(0, 0) - (imul(kx, ld(P_FEX)) + imul(ky, ld(P_FEY)) + imul(kz, ld(P_FEZ))) - (ph.mu * k2) * ld(P_Q);
    R[5] = imul(ky, ez) - imul(kz, ey) - (ph.eta * k2) * u[5];
    R[6] = imul(kz, ex) - imul(kx, ez) - (ph.eta * k2) * u[6];
    R[7] = imul(kx, ey) - imul(ky, ex) - (ph.eta * k2) * u[7];
}
// explicit update of one field of one mode: mode 1 Euler, 2 Adams-Bashforth 2 (R6)
__device__ __forceinline__ cd updated(int mode, double dt, cd u, cd R, cd ro) {
    cd inc;
    if (mode == 1) inc = R;
    else inc = mk(1.5 * R.x - 0.5 * ro.x, 1.5 * R.y - 0.5 * ro.y);
    return mk(u.x + dt * inc.x, u.y + dt * inc.y);
}

}  // namespace mhd

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

}  // namespace mhd

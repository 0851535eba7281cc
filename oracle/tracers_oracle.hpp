// oracle/tracers_oracle.hpp — CPU test oracle for the tracer particles of PAPER.md Sec. VI (L229-275).
// TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/oracle.h).  Shares no code with paper_1810_12707_b200/csrc.
//
// The paper's four steps (L268-272), one particle at a time, in the paper's order and notation:
//   1) grid index (i, j, k) of the bottom-left-front corner of the unit cell that holds particle m;
//   2) Eq. 20 (L251): cloud-in-cell interpolation of the grid magnetic field to the particle position, the weight
//      of each of the 8 corner grids being the volume of the OPPOSITE sub-cell of the unit cell; periodic wrap of
//      the corner indices (L255);
//   3) Eq. 21 (L259-265), Boris rotation with q = M = 1:
//        t = B_p dt/2 ;  s = 2 t/(1 + |t|^2) ;  v_d = v_t + v_t x t ;  v_{t+dt} = v_t + v_d x s ;
//   4) Eq. 22 (L266): x_{t+dt} = x_t + v_{t+dt} dt, wrapped back into [0, L) (L266 "periodic boundary condition
//      in the position of the tracers").
// Readings: T1 the weights of Eq. 20 are the sub-cell volumes divided by the cell
// volume (the factor "dt" and the repeated last terms printed in Eq. 20 are garbling: the weights must sum to 1 for
// a uniform field to be reproduced); T2 Eq. 21 is followed as printed (pure magnetic rotation, no electric field:
// "the time evolution of the tracers are fully governed by the magnetic fields", L241); T3 the initial velocity is
// the CIC interpolation of u = m/rho (L241 "evaluated from the velocity at the grid"); T4 positions are stored in
// [0, L), the cell index is floor(x / dx) evaluated in fp64.
// Written from the definitions (weights as cloud overlap with minimum-image distances, wrap by fmod) and kept
// deliberately unlike csrc/tracers.cu, so that GPU-vs-oracle parity can catch a misreading on either side.
// Everything is fp64 (the particle arithmetic is the paper's, Table I "double").
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>

namespace orc {

// minimum-image separation of two points on the periodic axis of length L: the representative of a - b in [-L/2, L/2]
inline double min_image(double a, double b, double L) {
    double d = std::fmod(a - b, L);
    if (d > 0.5 * L) d -= L;
    if (d < -0.5 * L) d += L;
    return d;
}

// steps 1-2, Eq. 20 for one scalar grid field g[z][y][x], written from the definition of cloud-in-cell weighting: the
// particle is a uniform cloud of the size of one cell, and a grid point receives the fraction of the cloud that
// overlaps its own cell, i.e. prod_axis max(0, 1 - |x_p - x_grid| / dx) with the periodic (minimum-image) distance.
// Only the grid points of the unit cell that holds the particle can have non-zero weight (step 1: its
// bottom-left-front corner is floor(x_p / dx), L249); they are visited corner by corner.
inline double cic(int N, double L, const double* g, const double x[3]) {
    const double dx = L / double(N);
    long long corner[3];
    for (int a = 0; a < 3; ++a) corner[a] = (long long)std::floor(x[a] / dx);
    double b = 0.0;
    for (int oz = 0; oz <= 1; ++oz)
        for (int oy = 0; oy <= 1; ++oy)
            for (int ox = 0; ox <= 1; ++ox) {
                const int off[3] = {ox, oy, oz};
                long long idx[3];
                double w = 1.0;
                for (int a = 0; a < 3; ++a) {
                    idx[a] = ((corner[a] + off[a]) % N + N) % N;                 // periodic wrap of the grid index (L255)
                    const double sep = std::fabs(min_image(x[a], double(idx[a]) * dx, L)) / dx;
                    w *= std::max(0.0, 1.0 - sep);
                }
                b += w * g[(std::int64_t(idx[2]) * N + idx[1]) * N + idx[0]];
            }
    return b;
}

// step 3, Eq. 21 (q = M = 1), with the vector algebra spelled out through a cross-product helper
inline void cross(const double a[3], const double b[3], double out[3]) {
    for (int c = 0; c < 3; ++c) out[c] = a[(c + 1) % 3] * b[(c + 2) % 3] - a[(c + 2) % 3] * b[(c + 1) % 3];
}
inline void boris(const double Bp[3], double dt, double v[3]) {
    double t[3], s[3], vxt[3], vd[3], vdxs[3];
    double t2 = 0.0;
    for (int c = 0; c < 3; ++c) { t[c] = 0.5 * dt * Bp[c]; t2 += t[c] * t[c]; }      // t = q B dt / 2M
    for (int c = 0; c < 3; ++c) s[c] = 2.0 * t[c] / (1.0 + t2);                       // s = 2 t / (1 + t^2)
    cross(v, t, vxt);
    for (int c = 0; c < 3; ++c) vd[c] = v[c] + vxt[c];                                // v_d = v_t + v_t x t
    cross(vd, s, vdxs);
    for (int c = 0; c < 3; ++c) v[c] += vdxs[c];                                      // v_{t+dt} = v_t + v_d x s
}

// Eq. 22 periodic wrap: the representative of x in [0, L)
inline double wrap(double x, double L) {
    double r = std::fmod(x, L);          // exact; sign of x
    if (r < 0.0) r += L;                 // may round to L when r = -tiny
    return r < L ? r : 0.0;              // L is the same point as 0
}

// steps 1-4 for np particles; B[c] are the three grid components; pos[c], vel[c] are updated in place
inline void tracers_push(int N, double L, double dt, const double* const B[3], long long np, double* const pos[3],
                         double* const vel[3]) {
    for (long long m = 0; m < np; ++m) {
        const double x[3] = {pos[0][m], pos[1][m], pos[2][m]};
        const double Bp[3] = {cic(N, L, B[0], x), cic(N, L, B[1], x), cic(N, L, B[2], x)};
        double v[3] = {vel[0][m], vel[1][m], vel[2][m]};
        boris(Bp, dt, v);
        for (int a = 0; a < 3; ++a) {
            vel[a][m] = v[a];
            pos[a][m] = wrap(x[a] + v[a] * dt, L);
        }
    }
}

// CIC interpolation of nf grid fields to np positions (used for the initial velocity, reading T3)
inline void tracers_interp(int N, double L, int nf, const double* const g[], long long np, const double* const pos[3],
                           double* const out[]) {
    for (long long m = 0; m < np; ++m) {
        const double x[3] = {pos[0][m], pos[1][m], pos[2][m]};
        for (int f = 0; f < nf; ++f) out[f][m] = cic(N, L, g[f], x);
    }
}

}  // namespace orc

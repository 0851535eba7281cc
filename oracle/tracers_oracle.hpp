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
// [0, L), the cell index is floor(x N/L) evaluated in fp64.
// Everything is fp64 (the particle arithmetic is the paper's, Table I "double").
#pragma once
#include <cmath>
#include <cstdint>

namespace orc {

struct Cell {           // step 1: corner indices (periodic) and the fractional position inside the cell
    int i0[3], i1[3];
    double f[3];
};

inline Cell locate(int N, double L, const double x[3]) {
    Cell c;
    const double inv_dx = double(N) / L;
    for (int a = 0; a < 3; ++a) {
        const double s = x[a] * inv_dx;
        const double fl = std::floor(s);
        c.f[a] = s - fl;
        long long i = (long long)fl % N;
        if (i < 0) i += N;
        c.i0[a] = int(i);
        c.i1[a] = int((i + 1) % N);
    }
    return c;
}

// step 2, Eq. 20 for one scalar grid field g[z][y][x]
inline double cic(int N, const double* g, const Cell& c) {
    const double fx = c.f[0], fy = c.f[1], fz = c.f[2];
    auto at = [&](int ix, int iy, int iz) { return g[(std::int64_t(iz) * N + iy) * N + ix]; };
    double b = 0.0;
    b += at(c.i0[0], c.i0[1], c.i0[2]) * ((1.0 - fx) * (1.0 - fy) * (1.0 - fz));
    b += at(c.i1[0], c.i0[1], c.i0[2]) * (fx * (1.0 - fy) * (1.0 - fz));
    b += at(c.i0[0], c.i1[1], c.i0[2]) * ((1.0 - fx) * fy * (1.0 - fz));
    b += at(c.i1[0], c.i1[1], c.i0[2]) * (fx * fy * (1.0 - fz));
    b += at(c.i0[0], c.i0[1], c.i1[2]) * ((1.0 - fx) * (1.0 - fy) * fz);
    b += at(c.i1[0], c.i0[1], c.i1[2]) * (fx * (1.0 - fy) * fz);
    b += at(c.i0[0], c.i1[1], c.i1[2]) * ((1.0 - fx) * fy * fz);
    b += at(c.i1[0], c.i1[1], c.i1[2]) * (fx * fy * fz);
    return b;
}

// step 3, Eq. 21 (q = M = 1)
inline void boris(const double Bp[3], double dt, double v[3]) {
    const double t[3] = {Bp[0] * (dt / 2.0), Bp[1] * (dt / 2.0), Bp[2] * (dt / 2.0)};
    const double t2 = t[0] * t[0] + t[1] * t[1] + t[2] * t[2];
    const double s[3] = {2.0 * t[0] / (1.0 + t2), 2.0 * t[1] / (1.0 + t2), 2.0 * t[2] / (1.0 + t2)};
    const double vd[3] = {v[0] + (v[1] * t[2] - v[2] * t[1]),
                          v[1] + (v[2] * t[0] - v[0] * t[2]),
                          v[2] + (v[0] * t[1] - v[1] * t[0])};
    const double vn[3] = {v[0] + (vd[1] * s[2] - vd[2] * s[1]),
                          v[1] + (vd[2] * s[0] - vd[0] * s[2]),
                          v[2] + (vd[0] * s[1] - vd[1] * s[0])};
    v[0] = vn[0]; v[1] = vn[1]; v[2] = vn[2];
}

inline double wrap(double x, double L) {
    x -= L * std::floor(x / L);
    if (x >= L) x -= L;      // x = -tiny gives L after rounding
    if (x < 0.0) x = 0.0;
    return x;
}

// steps 1-4 for np particles; B[c] are the three grid components; pos[c], vel[c] are updated in place
inline void tracers_push(int N, double L, double dt, const double* const B[3], long long np, double* const pos[3],
                         double* const vel[3]) {
    for (long long m = 0; m < np; ++m) {
        const double x[3] = {pos[0][m], pos[1][m], pos[2][m]};
        const Cell c = locate(N, L, x);
        const double Bp[3] = {cic(N, B[0], c), cic(N, B[1], c), cic(N, B[2], c)};
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
        const Cell c = locate(N, L, x);
        for (int f = 0; f < nf; ++f) out[f][m] = cic(N, g[f], c);
    }
}

}  // namespace orc

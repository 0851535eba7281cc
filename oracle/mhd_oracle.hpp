// oracle/mhd_oracle.hpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, obviously-correct CPU implementation of the one hot path this repository builds: the
// right-hand side and explicit (Adams-Bashforth) step of the 3-D compressible, viscous, resistive MHD
// equations on a triply periodic N^3 box, discretised pseudo-spectrally, as PAPER.md (arXiv 1810.12707,
// "G-MHD3D") defines them.  It shares no code, header, table or helper with the CUDA path under
// paper_1810_12707_b200/csrc/, and may be imported / linked / executed only by tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
//
// The method is not a fast route to some simpler closed form: the pseudo-spectral discretisation *is* the
// definition.  So this file follows the algorithm step by step in the paper's order and notation, every
// derivative by its own forward/inverse FFT pair, no fusion, no blocking, no shared transforms.
//
//   O0  transforms        own recursive radix-2 FFT, applied axis by axis on full complex N^3 arrays;
//                         direct O(N^6) DFT as the definition ("pseudo-spectral technique";
//                         L319-323 plan (Nz,Ny,Nx), D2Z forward / Z2D inverse; reading R7:
//                         forward unnormalised, inverse 1/N^3).
//   O1  operators         d~_j f = IFFT( M * i k_j * FFT f ),  lap~ f = IFFT( M * (-|k|^2) * FFT f ),
//                         M = 2/3-rule cubic mask max|n_j| <= floor(N/3)
//                         ("applied to calculate the spatial derivatives"; L27 dealiasing;
//                          DESIGN.md reading R5).
//   O2  state             conservative U = (rho, m=rho u, E, B), E = P/(gamma-1) + rho|u|^2/2 + |B|^2/2
//                         (PAPER.md:L85-86 with 1/8pi -> 1/2, reading R2; ideal-gas closure, reading R1).
//   O3  RHS               Eq. 17-19 for rho, m, B;  Eq. 12 (L96) for E in normalised
//                         units with the viscous work term matching mu lap u (reading R3);
//                         induction sign of Eq. 13 (L98, L110; reading R4).
//   O4  step              Adams-Bashforth 2 with forward-Euler start (reading R6).
//   O5  diagnostics       volume means "per grid", max|div~ B| (Eq. 9),
//                         shell spectra of sqrt(rho) u and B (L223; reading R8).
//
// Pins (tests/test_oracle_*.py, `-m "not gpu"`): direct DFT at 8^3 and numpy.fft (P1), exact derivatives and
// mask (P2), uniform state (P3), closed-form ABC / Orszag-Tang / shear / current-sheet RHS (P4-P7), the exact
// nonlinear circularly-polarised Alfven wave incl. AB2 order (P8), sound / fast-wave frequencies (P9),
// div B (P10), conservation (P11), AB2 recurrence (P12), brute-force DFT RHS at 8^3 (P13), closed-form
// diagnostics (P14).  No function of this file is "parity unpinned".
//
// Templated on the real type (double / long double) so the fp64 noise floor of the RHS can be measured
// (criterion 3).
#pragma once

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <stdexcept>
#include <vector>

namespace orc {

template <class T> using cplx = std::complex<T>;
template <class T> using rfield = std::vector<T>;
template <class T> using cfield = std::vector<cplx<T>>;

template <class T> inline T pi_v() { return std::acos(T(-1)); }

// ------------------------------------------------------------------------------------------------
// O0. transforms
// ------------------------------------------------------------------------------------------------

// exp(-2 pi i j / n), j = 0..n-1, each entry evaluated directly (no recurrences).
template <class T> std::vector<cplx<T>> unit_roots(int n) {
    std::vector<cplx<T>> w(n);
    for (int j = 0; j < n; ++j) {
        T a = T(2) * pi_v<T>() * T(j) / T(n);
        w[j] = cplx<T>(std::cos(a), -std::sin(a));
    }
    return w;
}

// Recursive radix-2 decimation-in-time FFT of length n (power of two), unnormalised.
//   out[k] = sum_j in[j*stride] * exp(sign * 2 pi i j k / n),  sign = -1 forward, +1 inverse.
// `w` holds exp(-2 pi i j / nroot), nroot >= n, wstep = nroot / n.
template <class T>
void fft_rec(const cplx<T>* in, int stride, cplx<T>* out, int n, const cplx<T>* w, int wstep, int sign) {
    if (n == 1) { out[0] = in[0]; return; }
    const int h = n / 2;
    fft_rec(in, 2 * stride, out, h, w, 2 * wstep, sign);               // even samples -> out[0..h)
    fft_rec(in + stride, 2 * stride, out + h, h, w, 2 * wstep, sign);  // odd samples  -> out[h..n)
    for (int k = 0; k < h; ++k) {
        cplx<T> tw = w[k * wstep];
        if (sign > 0) tw = std::conj(tw);
        const cplx<T> e = out[k], o = tw * out[k + h];
        out[k] = e + o;
        out[k + h] = e - o;
    }
}

// 3-D transform of a full complex N^3 array a[z][y][x] (x fastest), axis by axis, in place.
// sign=-1: F[n] = sum_x f[x] exp(-2 pi i n.x/N) (unnormalised); sign=+1: same with +, times 1/N^3.
template <class T> void fft3(cfield<T>& a, int N, int sign) {
    const std::vector<cplx<T>> w = unit_roots<T>(N);
    const std::int64_t N2 = std::int64_t(N) * N;
    const std::int64_t strides[3] = {1, N, N2};  // x, y, z
    for (int axis = 0; axis < 3; ++axis) {
        const std::int64_t s = strides[axis];
#pragma omp parallel
        {
            std::vector<cplx<T>> buf(N), res(N);
#pragma omp for schedule(static)
            for (std::int64_t p = 0; p < N2; ++p) {
                // the p-th pencil along `axis`: the two other indices enumerate p
                std::int64_t base;
                if (axis == 0) base = p * N;                         // (z,y) -> z*N^2 + y*N
                else if (axis == 1) base = (p / N) * N2 + (p % N);   // (z,x)
                else base = p;                                       // (y,x)
                for (int j = 0; j < N; ++j) buf[j] = a[base + j * s];
                fft_rec(buf.data(), 1, res.data(), N, w.data(), 1, sign);
                for (int j = 0; j < N; ++j) a[base + j * s] = res[j];
            }
        }
    }
    if (sign > 0) {
        const T inv = T(1) / (T(N) * T(N) * T(N));
        for (auto& v : a) v *= inv;
    }
}

// The definition: direct O(N^6) DFT, every phase evaluated on its own (no table, no FFT).
template <class T> void dft3_direct(const cfield<T>& in, cfield<T>& out, int N, int sign) {
    const std::int64_t N3 = std::int64_t(N) * N * N;
    out.assign(N3, cplx<T>(0));
    const T two_pi = T(2) * pi_v<T>();
#pragma omp parallel for schedule(static)
    for (std::int64_t q = 0; q < N3; ++q) {
        const int kz = int(q / (std::int64_t(N) * N)), ky = int((q / N) % N), kx = int(q % N);
        cplx<T> acc(0);
        for (int z = 0; z < N; ++z)
            for (int y = 0; y < N; ++y)
                for (int x = 0; x < N; ++x) {
                    const int m = (kx * x + ky * y + kz * z) % N;  // exact integer phase reduction
                    const T ang = two_pi * T(m) / T(N);
                    const cplx<T> ph(std::cos(ang), T(sign) * std::sin(ang));
                    acc += in[(std::int64_t(z) * N + y) * N + x] * ph;
                }
        out[q] = (sign > 0) ? acc / (T(N) * T(N) * T(N)) : acc;
    }
}

// ------------------------------------------------------------------------------------------------
// diagnostics record (layout mirrored, not shared, by include/mhd.h)
// ------------------------------------------------------------------------------------------------
struct Diag {
    double t;
    long long step;
    double ke, me, ie, mass, mom[3], etot, max_divb, rho_min, p_min;
};

// ------------------------------------------------------------------------------------------------
// the solver
// ------------------------------------------------------------------------------------------------
template <class T> class Solver {
public:
    enum { RHO = 0, MX, MY, MZ, EN, BX, BY, BZ, NF };

    Solver(int N_, double L_, double gamma_, double mu_, double eta_, double dt_)
        : N(N_), L(T(L_)), gamma(T(gamma_)), mu(T(mu_)), eta(T(eta_)), dt(T(dt_)) {
        if (N < 4 || (N & (N - 1))) throw std::invalid_argument("N must be a power of two >= 4");
        N3 = std::int64_t(N) * N * N;
        kc = N / 3;
        for (auto& f : U) f.assign(N3, T(0));
        k0 = T(2) * pi_v<T>() / L;
    }

    int N;
    std::int64_t N3;
    int kc;                 // 2/3-rule cut-off, floor(N/3)
    T L, gamma, mu, eta, dt, k0;
    T time = T(0);
    long long nstep = 0;
    // Equation-set variants of the paper (readings V1-V3):
    T cs2 = T(0);      // > 0: barotropic closure P = C_s^2 rho of Eq. 5 / Eq. 18 (L63, L192); E is then not evolved
    T f0 = T(0);       // amplitude of the ABC forcing rho f of Eq. 18 / L215, f = f0 (sin kz + cos ky, sin kx + cos kz, sin ky + cos kx)
    int kf = 1;        // its integer mode number k_f (k = k_f 2 pi/L)
    int stress = 0;    // 1: the viscous terms of Eq. 11-12 (L92-96): + div(2 nu rho S) in the momentum equation and the energy
                       //    flux -2 nu rho u.S, with S of Eq. 3-4 (L57-61) and nu = the `mu` parameter, instead of R3's mu lap u
    int evolve = 3;    // bit 0: Eq. 17-18 (+ energy) evolve; bit 1: Eq. 19 evolves ("turn off" of L199 / L205)
    bool use_direct_dft = false;   // P13: substitute the O(N^6) definition for the FFT
    bool have_fields = false;
    rfield<T> U[NF];        // conservative state in real space
    rfield<T> Rold[NF];     // previous RHS (AB2 history)
    bool have_old = false;

    // mode number of array index i: n(i) = i for i <= N/2, i-N otherwise
    int mode(int i) const { return i <= N / 2 ? i : i - N; }
    // M(n) = 1 iff max(|nx|,|ny|,|nz|) <= kc   (reading R5: cubic 2/3-rule truncation)
    bool mask(int nx, int ny, int nz) const {
        return std::abs(nx) <= kc && std::abs(ny) <= kc && std::abs(nz) <= kc;
    }

    void forward(cfield<T>& a) const {
        if (use_direct_dft) { cfield<T> o; dft3_direct(a, o, N, -1); a.swap(o); } else fft3(a, N, -1);
    }
    void inverse(cfield<T>& a) const {
        if (use_direct_dft) { cfield<T> o; dft3_direct(a, o, N, +1); a.swap(o); } else fft3(a, N, +1);
    }

    // --------------------------------------------------------------------------------------------
    // O1. the one dealiased operator family.  op = 0,1,2: d/dx, d/dy, d/dz; 3: Laplacian; 4: projection M.
    // --------------------------------------------------------------------------------------------
    void apply(const rfield<T>& f, int op, rfield<T>& out) const {
        cfield<T> a(N3);
        for (std::int64_t i = 0; i < N3; ++i) a[i] = cplx<T>(f[i], T(0));
        forward(a);
        for (int iz = 0; iz < N; ++iz)
            for (int iy = 0; iy < N; ++iy)
                for (int ix = 0; ix < N; ++ix) {
                    const int nx = mode(ix), ny = mode(iy), nz = mode(iz);
                    cplx<T>& v = a[(std::int64_t(iz) * N + iy) * N + ix];
                    if (!mask(nx, ny, nz)) { v = cplx<T>(0); continue; }
                    const T kx = k0 * T(nx), ky = k0 * T(ny), kz = k0 * T(nz);
                    switch (op) {
                        case 0: v *= cplx<T>(T(0), kx); break;
                        case 1: v *= cplx<T>(T(0), ky); break;
                        case 2: v *= cplx<T>(T(0), kz); break;
                        case 3: v *= -(kx * kx + ky * ky + kz * kz); break;
                        default: break;
                    }
                }
        inverse(a);
        out.resize(N3);
        for (std::int64_t i = 0; i < N3; ++i) out[i] = a[i].real();
    }
    rfield<T> d(const rfield<T>& f, int axis) const { rfield<T> o; apply(f, axis, o); return o; }
    rfield<T> lap(const rfield<T>& f) const { rfield<T> o; apply(f, 3, o); return o; }
    rfield<T> project(const rfield<T>& f) const { rfield<T> o; apply(f, 4, o); return o; }

    // --------------------------------------------------------------------------------------------
    // O2. state in / out.  kind 0 = conservative (rho,mx,my,mz,E,Bx,By,Bz), 1 = primitive (rho,u,P,B)
    // --------------------------------------------------------------------------------------------
    void set_fields(int kind, const double* const f[NF]) {
        rfield<T> in[NF];
        for (int c = 0; c < NF; ++c) {
            in[c].resize(N3);
            for (std::int64_t i = 0; i < N3; ++i) in[c][i] = T(f[c][i]);
        }
        if (kind == 1) {
            for (std::int64_t i = 0; i < N3; ++i) {
                const T rho = in[0][i], ux = in[1][i], uy = in[2][i], uz = in[3][i], P = in[4][i];
                const T bx = in[5][i], by = in[6][i], bz = in[7][i];
                in[MX][i] = rho * ux; in[MY][i] = rho * uy; in[MZ][i] = rho * uz;
                // E = rho eps_int + rho|u|^2/2 + |B|^2/2   (normalised units)
                in[EN][i] = P / (gamma - T(1)) + T(0.5) * rho * (ux * ux + uy * uy + uz * uz)
                          + T(0.5) * (bx * bx + by * by + bz * bz);
            }
        }
        for (int c = 0; c < NF; ++c) U[c] = project(in[c]);   // U <- IFFT(M FFT U)   (reading R5)
        time = T(0); nstep = 0; have_old = false; have_fields = true;
    }

    void get_fields(int kind, double* const out[NF]) const {
        for (std::int64_t i = 0; i < N3; ++i) {
            if (kind == 0) { for (int c = 0; c < NF; ++c) out[c][i] = double(U[c][i]); continue; }
            const T rho = U[RHO][i], ux = U[MX][i] / rho, uy = U[MY][i] / rho, uz = U[MZ][i] / rho;
            const T bx = U[BX][i], by = U[BY][i], bz = U[BZ][i];
            const T P = (gamma - T(1)) * (U[EN][i] - T(0.5) * (U[MX][i] * ux + U[MY][i] * uy + U[MZ][i] * uz)
                                          - T(0.5) * (bx * bx + by * by + bz * bz));
            out[0][i] = double(rho); out[1][i] = double(ux); out[2][i] = double(uy); out[3][i] = double(uz);
            out[4][i] = double(P); out[5][i] = double(bx); out[6][i] = double(by); out[7][i] = double(bz);
        }
    }

    // --------------------------------------------------------------------------------------------
    // O3. right-hand side  R = dU/dt.  If phi/dsc are given they receive, per field, the L2 norm of the
    //     stacked real-space flux and the diffusion scale (SURVEY.md §8(c)-T backward-error criterion).
    // --------------------------------------------------------------------------------------------
    void rhs(const rfield<T> (&S)[NF], rfield<T> (&R)[NF], double* phi = nullptr, double* dsc = nullptr) const {
        const rfield<T>&rho = S[RHO], &mx = S[MX], &my = S[MY], &mz = S[MZ], &E = S[EN];
        const rfield<T>* B[3] = {&S[BX], &S[BY], &S[BZ]};
        const rfield<T>* m[3] = {&mx, &my, &mz};

        // primitive recovery: u = m/rho, P = (gamma-1)(E - m.u/2 - |B|^2/2), Pt = P + |B|^2/2  (L85-86)
        rfield<T> u[3], Pt(N3), q(N3);
        for (auto& c : u) c.resize(N3);
        for (std::int64_t i = 0; i < N3; ++i) {
            for (int c = 0; c < 3; ++c) u[c][i] = (*m[c])[i] / rho[i];
            const T b2 = (*B[0])[i] * (*B[0])[i] + (*B[1])[i] * (*B[1])[i] + (*B[2])[i] * (*B[2])[i];
            const T mu_dot = mx[i] * u[0][i] + my[i] * u[1][i] + mz[i] * u[2][i];
            const T P = cs2 > T(0) ? cs2 * rho[i] : (gamma - T(1)) * (E[i] - T(0.5) * mu_dot - T(0.5) * b2);
            Pt[i] = P + T(0.5) * b2;
            q[i] = T(0.5) * (u[0][i] * u[0][i] + u[1][i] * u[1][i] + u[2][i] * u[2][i]);
        }

        // J = curl~ B   (Eq. 6 without c/4pi)
        rfield<T> J[3];
        {
            const rfield<T> dyBz = d(*B[2], 1), dzBy = d(*B[1], 2);
            const rfield<T> dzBx = d(*B[0], 2), dxBz = d(*B[2], 0);
            const rfield<T> dxBy = d(*B[1], 0), dyBx = d(*B[0], 1);
            for (auto& c : J) c.resize(N3);
            for (std::int64_t i = 0; i < N3; ++i) {
                J[0][i] = dyBz[i] - dzBy[i];
                J[1][i] = dzBx[i] - dxBz[i];
                J[2][i] = dxBy[i] - dyBx[i];
            }
        }

        std::vector<double> phi2(NF, 0.0);
        auto accum_phi = [&](int f, const rfield<T>& flux) {
            if (!phi) return;
            long double s = 0;
            for (std::int64_t i = 0; i < N3; ++i) s += (long double)flux[i] * (long double)flux[i];
            phi2[f] += double(s);
        };
        auto l2 = [&](const rfield<T>& a) {
            long double s = 0;
            for (std::int64_t i = 0; i < N3; ++i) s += (long double)a[i] * (long double)a[i];
            return double(std::sqrt(s));
        };

        // Eq. 17:  d rho/dt = - d_j m_j
        {
            R[RHO].assign(N3, T(0));
            for (int j = 0; j < 3; ++j) {
                const rfield<T> dj = d(*m[j], j);
                accum_phi(RHO, *m[j]);
                for (std::int64_t i = 0; i < N3; ++i) R[RHO][i] -= dj[i];
            }
        }

        // Eq. 18:  d m_i/dt = - d_j ( m_i u_j + Pt delta_ij - B_i B_j ) + mu lap u_i
        for (int c = 0; c < 3; ++c) {
            rfield<T>& out = R[MX + c];
            out.assign(N3, T(0));
            for (int j = 0; j < 3; ++j) {
                rfield<T> flux(N3);
                for (std::int64_t i = 0; i < N3; ++i)
                    flux[i] = (*m[c])[i] * u[j][i] + (c == j ? Pt[i] : T(0)) - (*B[c])[i] * (*B[j])[i];
                const rfield<T> dj = d(flux, j);
                accum_phi(MX + c, flux);
                for (std::int64_t i = 0; i < N3; ++i) out[i] -= dj[i];
            }
            if (!stress) {
                const rfield<T> lu = lap(u[c]);
                for (std::int64_t i = 0; i < N3; ++i) out[i] += mu * lu[i];
            }
        }

        // Eq. 12:  dE/dt = - d_j ( (E+Pt) u_j - (u.B) B_j - eta (B x J)_j ) + mu lap (|u|^2/2)
        {
            rfield<T>& out = R[EN];
            out.assign(N3, T(0));
            for (int j = 0; j < 3; ++j) {
                const int a = (j + 1) % 3, b = (j + 2) % 3;
                rfield<T> flux(N3);
                for (std::int64_t i = 0; i < N3; ++i) {
                    const T udotB = u[0][i] * (*B[0])[i] + u[1][i] * (*B[1])[i] + u[2][i] * (*B[2])[i];
                    const T BxJ = (*B[a])[i] * J[b][i] - (*B[b])[i] * J[a][i];
                    flux[i] = (E[i] + Pt[i]) * u[j][i] - udotB * (*B[j])[i] - eta * BxJ;
                }
                const rfield<T> dj = d(flux, j);
                accum_phi(EN, flux);
                for (std::int64_t i = 0; i < N3; ++i) out[i] -= dj[i];
            }
            if (!stress) {
                const rfield<T> lq = lap(q);
                for (std::int64_t i = 0; i < N3; ++i) out[i] += mu * lq[i];
            }
        }

        // Eq. 11-12 viscous terms (variant `stress`): S_ij = (d_i u_j + d_j u_i)/2 - delta_ij theta/3, theta = div u (Eq. 3-4);
        // momentum + d_j (2 nu rho S_ij); energy - d_j ( -2 nu rho u_i S_ij ) = + d_j (2 nu rho u_i S_ij)
        if (stress) {
            rfield<T> du[3][3];                         // du[i][j] = d_i u_j
            for (int i = 0; i < 3; ++i)
                for (int j = 0; j < 3; ++j) du[i][j] = d(u[j], i);
            rfield<T> V[3][3];                          // 2 nu rho S_ij
            for (int i = 0; i < 3; ++i)
                for (int j = 0; j < 3; ++j) V[i][j].resize(N3);
            for (std::int64_t p = 0; p < N3; ++p) {
                const T theta = du[0][0][p] + du[1][1][p] + du[2][2][p];
                for (int i = 0; i < 3; ++i)
                    for (int j = 0; j < 3; ++j) {
                        const T Sij = T(0.5) * (du[i][j][p] + du[j][i][p]) - (i == j ? theta / T(3) : T(0));
                        V[i][j][p] = T(2) * mu * rho[p] * Sij;
                    }
            }
            for (int i = 0; i < 3; ++i)
                for (int j = 0; j < 3; ++j) {
                    const rfield<T> dj = d(V[i][j], j);
                    for (std::int64_t p = 0; p < N3; ++p) R[MX + i][p] += dj[p];
                }
            for (int j = 0; j < 3; ++j) {
                rfield<T> w(N3);
                for (std::int64_t p = 0; p < N3; ++p) w[p] = u[0][p] * V[0][j][p] + u[1][p] * V[1][j][p] + u[2][p] * V[2][j][p];
                const rfield<T> dj = d(w, j);
                for (std::int64_t p = 0; p < N3; ++p) R[EN][p] += dj[p];
            }
        }

        // Eq. 19 / 13:  dB/dt = curl~ (u x B) + eta lap B, component form of PAPER.md:L110
        {
            rfield<T> exy(N3), exz(N3), eyz(N3);   // ux By - uy Bx,  ux Bz - uz Bx,  uy Bz - uz By
            for (std::int64_t i = 0; i < N3; ++i) {
                exy[i] = u[0][i] * (*B[1])[i] - u[1][i] * (*B[0])[i];
                exz[i] = u[0][i] * (*B[2])[i] - u[2][i] * (*B[0])[i];
                eyz[i] = u[1][i] * (*B[2])[i] - u[2][i] * (*B[1])[i];
            }
            const rfield<T> dy_exy = d(exy, 1), dz_exz = d(exz, 2);
            const rfield<T> dx_exy = d(exy, 0), dz_eyz = d(eyz, 2);
            const rfield<T> dx_exz = d(exz, 0), dy_eyz = d(eyz, 1);
            const rfield<T> lbx = lap(*B[0]), lby = lap(*B[1]), lbz = lap(*B[2]);
            for (int c = 0; c < 3; ++c) R[BX + c].assign(N3, T(0));
            for (std::int64_t i = 0; i < N3; ++i) {
                R[BX][i] = dy_exy[i] + dz_exz[i] + eta * lbx[i];
                R[BY][i] = -dx_exy[i] + dz_eyz[i] + eta * lby[i];
                R[BZ][i] = -dx_exz[i] - dy_eyz[i] + eta * lbz[i];
            }
            accum_phi(BX, exy); accum_phi(BX, exz);
            accum_phi(BY, exy); accum_phi(BY, eyz);
            accum_phi(BZ, exz); accum_phi(BZ, eyz);
        }

        // Eq. 18 forcing rho f (L192, L215) and its work m.f in the energy equation (reading V1); like every product
        // it is dealias-projected (operator family O1, op 4)
        if (f0 != T(0)) {
            rfield<T> f[3];
            for (auto& c : f) c.resize(N3);
            const T kk = k0 * T(kf), dx = L / T(N);
            for (int iz = 0; iz < N; ++iz)
                for (int iy = 0; iy < N; ++iy)
                    for (int ix = 0; ix < N; ++ix) {
                        const std::int64_t i = (std::int64_t(iz) * N + iy) * N + ix;
                        const T x = dx * T(ix), y = dx * T(iy), z = dx * T(iz);
                        f[0][i] = f0 * (std::sin(kk * z) + std::cos(kk * y));
                        f[1][i] = f0 * (std::sin(kk * x) + std::cos(kk * z));
                        f[2][i] = f0 * (std::sin(kk * y) + std::cos(kk * x));
                    }
            rfield<T> work(N3, T(0));
            for (int c = 0; c < 3; ++c) {
                rfield<T> prod(N3);
                for (std::int64_t i = 0; i < N3; ++i) { prod[i] = rho[i] * f[c][i]; work[i] += (*m[c])[i] * f[c][i]; }
                const rfield<T> pr = project(prod);
                for (std::int64_t i = 0; i < N3; ++i) R[MX + c][i] += pr[i];
            }
            const rfield<T> pw = project(work);
            for (std::int64_t i = 0; i < N3; ++i) R[EN][i] += pw[i];
        }
        if (cs2 > T(0)) R[EN].assign(N3, T(0));                              // barotropic: no energy equation
        if (!(evolve & 1)) for (int c = RHO; c <= EN; ++c) R[c].assign(N3, T(0));
        if (!(evolve & 2)) for (int c = BX; c <= BZ; ++c) R[c].assign(N3, T(0));

        if (phi) for (int f = 0; f < NF; ++f) phi[f] = std::sqrt(phi2[f]);
        if (dsc) {
            dsc[RHO] = 0.0;
            for (int c = 0; c < 3; ++c) dsc[MX + c] = double(mu) * l2(u[c]);
            dsc[EN] = double(mu) * l2(q);
            for (int c = 0; c < 3; ++c) dsc[BX + c] = double(eta) * l2(*B[c]);
        }
    }

    // --------------------------------------------------------------------------------------------
    // O4. Adams-Bashforth 2, forward-Euler start (reading R6)
    // --------------------------------------------------------------------------------------------
    // integrator: 0 = Adams-Bashforth 2 (above); 1 = classical Runge-Kutta 4; 2 = predictor-corrector (Heun):
    // U* = U + dt R(U), U+ = U + dt/2 (R(U) + R(U*)) — the paper's other two time solvers (Table I)
    int integrator = 0;

    void axpy(rfield<T> (&y)[NF], const rfield<T> (&base)[NF], T a, const rfield<T> (&x)[NF]) const {   // y = base + a x
        for (int c = 0; c < NF; ++c) {
            y[c].resize(N3);
            for (std::int64_t i = 0; i < N3; ++i) y[c][i] = base[c][i] + a * x[c][i];
        }
    }
    void step_rk4() {
        rfield<T> k1[NF], k2[NF], k3[NF], k4[NF], S[NF];
        rhs(U, k1);
        axpy(S, U, T(0.5) * dt, k1); rhs(S, k2);
        axpy(S, U, T(0.5) * dt, k2); rhs(S, k3);
        axpy(S, U, dt, k3);          rhs(S, k4);
        for (int c = 0; c < NF; ++c)
            for (std::int64_t i = 0; i < N3; ++i)
                U[c][i] += dt * (k1[c][i] / T(6) + k2[c][i] / T(3) + k3[c][i] / T(3) + k4[c][i] / T(6));
    }
    void step_heun() {
        rfield<T> r0[NF], r1[NF], S[NF];
        rhs(U, r0);
        axpy(S, U, dt, r0);          // predictor
        rhs(S, r1);
        for (int c = 0; c < NF; ++c)
            for (std::int64_t i = 0; i < N3; ++i) U[c][i] += T(0.5) * dt * (r0[c][i] + r1[c][i]);
    }

    void step(int nsteps) {
        for (int s = 0; s < nsteps && integrator != 0; ++s) {
            if (integrator == 1) step_rk4(); else step_heun();
            ++nstep;
            time = T(nstep) * dt;
        }
        if (integrator != 0) return;
        for (int s = 0; s < nsteps; ++s) {
            rfield<T> R[NF];
            rhs(U, R);
            for (int c = 0; c < NF; ++c) {
                if (!have_old) {
                    for (std::int64_t i = 0; i < N3; ++i) U[c][i] += dt * R[c][i];
                } else {
                    for (std::int64_t i = 0; i < N3; ++i)
                        U[c][i] += dt * (T(1.5) * R[c][i] - T(0.5) * Rold[c][i]);
                }
                Rold[c].swap(R[c]);
            }
            have_old = true;
            ++nstep;
            time = T(nstep) * dt;
        }
    }

    // --------------------------------------------------------------------------------------------
    // O5. diagnostics.  nspec must be ceil(sqrt(3) N/2) + 1 when spectra are requested.
    // --------------------------------------------------------------------------------------------
    int nspec() const { return int(std::ceil(std::sqrt(3.0) * N / 2.0)) + 1; }

    void diagnostics(Diag& dg, double* spec_kin, double* spec_mag) const {
        // serial sums in fixed order, accumulated in long double so that the mean of N^3 terms does not
        // carry a sqrt(N^3)-ulp random walk (the per-point arithmetic stays in T)
        typedef long double A;
        A ke = 0, me = 0, ie = 0, mass = 0, mom[3] = {0, 0, 0}, etot = 0;
        T rho_min = U[RHO][0], p_min = T(0);
        bool first = true;
        for (std::int64_t i = 0; i < N3; ++i) {
            const T rho = U[RHO][i];
            const T ux = U[MX][i] / rho, uy = U[MY][i] / rho, uz = U[MZ][i] / rho;
            const T b2 = U[BX][i] * U[BX][i] + U[BY][i] * U[BY][i] + U[BZ][i] * U[BZ][i];
            const T k = T(0.5) * (U[MX][i] * ux + U[MY][i] * uy + U[MZ][i] * uz);
            const T P = (gamma - T(1)) * (U[EN][i] - k - T(0.5) * b2);
            ke += k; me += T(0.5) * b2; ie += P / (gamma - T(1)); mass += rho; etot += U[EN][i];
            mom[0] += U[MX][i]; mom[1] += U[MY][i]; mom[2] += U[MZ][i];
            rho_min = std::min(rho_min, rho);
            p_min = first ? P : std::min(p_min, P);
            first = false;
        }
        const A inv = A(1) / A(N3);
        dg.t = double(time); dg.step = nstep;
        dg.ke = double(ke * inv); dg.me = double(me * inv); dg.ie = double(ie * inv);
        dg.mass = double(mass * inv); dg.etot = double(etot * inv);
        for (int c = 0; c < 3; ++c) dg.mom[c] = double(mom[c] * inv);
        dg.rho_min = double(rho_min); dg.p_min = double(p_min);

        // max | d~x Bx + d~y By + d~z Bz |   (Eq. 9)
        {
            const rfield<T> a = d(U[BX], 0), b = d(U[BY], 1), c = d(U[BZ], 2);
            T mx_ = 0;
            for (std::int64_t i = 0; i < N3; ++i) mx_ = std::max(mx_, std::abs(a[i] + b[i] + c[i]));
            dg.max_divb = double(mx_);
        }

        if (spec_kin || spec_mag) {
            const int ns = nspec();
            // S(K) = sum_{n: floor(|n|+1/2)=K}  1/2 sum_c |w^_c(n)|^2 / N^6   over the FULL n-cube
            auto shell = [&](const rfield<T> (&w)[3], double* out) {
                std::vector<long double> S(ns, 0.0L);
                for (int c = 0; c < 3; ++c) {
                    cfield<T> a(N3);
                    for (std::int64_t i = 0; i < N3; ++i) a[i] = cplx<T>(w[c][i], T(0));
                    forward(a);
                    for (int iz = 0; iz < N; ++iz)
                        for (int iy = 0; iy < N; ++iy)
                            for (int ix = 0; ix < N; ++ix) {
                                const int nx = mode(ix), ny = mode(iy), nz = mode(iz);
                                const double r = std::sqrt(double(nx * nx + ny * ny + nz * nz));
                                const int K = int(std::floor(r + 0.5));
                                S[K] += T(0.5) * std::norm(a[(std::int64_t(iz) * N + iy) * N + ix]);
                            }
                }
                const long double n6 = (long double)N3 * (long double)N3;
                for (int K = 0; K < ns; ++K) out[K] = double(S[K] / n6);
            };
            if (spec_kin) {
                rfield<T> w[3];
                for (int c = 0; c < 3; ++c) {
                    w[c].resize(N3);
                    for (std::int64_t i = 0; i < N3; ++i) w[c][i] = U[MX + c][i] / std::sqrt(U[RHO][i]);
                }
                shell(w, spec_kin);
            }
            if (spec_mag) {
                rfield<T> w[3] = {U[BX], U[BY], U[BZ]};
                shell(w, spec_mag);
            }
        }
    }
};

}  // namespace orc

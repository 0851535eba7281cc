// oracle/oracle_capi.cpp — C interface of the CPU test oracle (TEST INFRASTRUCTURE, NOT THE PRODUCT).
// See oracle/oracle.h and oracle/mhd_oracle.hpp.  Build: oracle/build_oracle.py (g++ -O2 -fopenmp -shared).
#include "oracle.h"
#include "mhd_oracle.hpp"
#include "tracers_oracle.hpp"

#include <algorithm>
#include <memory>
#include <vector>
#include <string>
#ifdef _OPENMP
#include <omp.h>
#endif

struct orc_ctx {
    int precision;
    std::unique_ptr<orc::Solver<double>> d;
    std::unique_ptr<orc::Solver<long double>> ld;
    long long np = 0;                       // attached tracers (fp64 whatever the field precision)
    std::vector<double> tpos[3], tvel[3];
};

static thread_local std::string g_err;

template <class F> static int guarded(F&& f) {
    try { f(); return 0; }
    catch (const std::exception& e) { g_err = e.what(); return -1; }
    catch (...) { g_err = "unknown exception"; return -1; }
}

#define DISPATCH(c, expr) do { if ((c)->precision == 0) { auto& S = *(c)->d; expr; } else { auto& S = *(c)->ld; expr; } } while (0)

template <class T> static void rhs_out(orc::Solver<T>& S, double* const out[8], double* phi, double* dsc) {
    if (!S.have_fields) throw std::runtime_error("no fields set");
    orc::rfield<T> R[8];
    S.rhs(S.U, R, phi, dsc);
    for (int c = 0; c < 8; ++c)
        for (std::int64_t i = 0; i < S.N3; ++i) out[c][i] = double(R[c][i]);
}

template <class T> static void apply_out(orc::Solver<T>& S, int op, const double* in, double* out) {
    orc::rfield<T> f(S.N3), o;
    for (std::int64_t i = 0; i < S.N3; ++i) f[i] = T(in[i]);
    S.apply(f, op, o);
    for (std::int64_t i = 0; i < S.N3; ++i) out[i] = double(o[i]);
}

template <class T> static void transform(int N, int sign, bool direct, const double* in, double* out) {
    const std::int64_t N3 = std::int64_t(N) * N * N;
    orc::cfield<T> a(N3), o;
    for (std::int64_t i = 0; i < N3; ++i) a[i] = orc::cplx<T>(T(in[2 * i]), T(in[2 * i + 1]));
    if (direct) { orc::dft3_direct(a, o, N, sign); a.swap(o); } else orc::fft3(a, N, sign);
    for (std::int64_t i = 0; i < N3; ++i) { out[2 * i] = double(a[i].real()); out[2 * i + 1] = double(a[i].imag()); }
}

template <class T> static void grid_B_u(const orc::Solver<T>& S, std::vector<double> (&B)[3], std::vector<double> (*u)[3]) {
    for (int a = 0; a < 3; ++a) {
        B[a].resize(S.N3);
        if (u) (*u)[a].resize(S.N3);
        for (std::int64_t i = 0; i < S.N3; ++i) {
            B[a][i] = double(S.U[5 + a][i]);
            if (u) (*u)[a][i] = double(S.U[1 + a][i] / S.U[0][i]);
        }
    }
}
template <class T> static void step_with_tracers(orc_ctx* c, orc::Solver<T>& S, int nsteps) {
    if (!S.have_fields) throw std::runtime_error("no fields set");
    if (c->np == 0) { S.step(nsteps); return; }
    for (int s = 0; s < nsteps; ++s) {
        std::vector<double> B[3];
        grid_B_u(S, B, nullptr);
        const double* Bp[3] = {B[0].data(), B[1].data(), B[2].data()};
        double* pos[3] = {c->tpos[0].data(), c->tpos[1].data(), c->tpos[2].data()};
        double* vel[3] = {c->tvel[0].data(), c->tvel[1].data(), c->tvel[2].data()};
        orc::tracers_push(S.N, double(S.L), double(S.dt), Bp, c->np, pos, vel);   // B at t_n, then the fields advance
        S.step(1);
    }
}
template <class T> static void tracers_attach(orc_ctx* c, orc::Solver<T>& S, long long np, const double* const vel[3]) {
    for (int a = 0; a < 3; ++a)
        for (long long m = 0; m < np; ++m) c->tpos[a][m] = orc::wrap(c->tpos[a][m], double(S.L));
    if (vel) { for (int a = 0; a < 3; ++a) c->tvel[a].assign(vel[a], vel[a] + np); return; }
    if (!S.have_fields) throw std::runtime_error("no fields set");
    std::vector<double> B[3], u[3];
    grid_B_u(S, B, &u);
    const double* g[3] = {u[0].data(), u[1].data(), u[2].data()};
    const double* p[3] = {c->tpos[0].data(), c->tpos[1].data(), c->tpos[2].data()};
    double* o[3] = {c->tvel[0].data(), c->tvel[1].data(), c->tvel[2].data()};
    orc::tracers_interp(S.N, double(S.L), 3, g, np, p, o);
}

extern "C" {

int orc_create(orc_ctx** out, int N, double L, double gamma, double mu, double eta, double dt, int precision) {
    return guarded([&] {
        if (!out) throw std::invalid_argument("null out");
        if (!(L > 0) || !(gamma > 1) || mu < 0 || eta < 0 || !(dt > 0)) throw std::invalid_argument("bad parameter");
        auto c = std::make_unique<orc_ctx>();
        c->precision = precision ? 1 : 0;
        if (c->precision == 0) c->d = std::make_unique<orc::Solver<double>>(N, L, gamma, mu, eta, dt);
        else c->ld = std::make_unique<orc::Solver<long double>>(N, L, gamma, mu, eta, dt);
        *out = c.release();
    });
}

int orc_destroy(orc_ctx* c) { delete c; return 0; }
const char* orc_last_error(void) { return g_err.c_str(); }

void orc_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
int orc_get_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

int orc_use_direct_dft(orc_ctx* c, int on) { return guarded([&] { DISPATCH(c, S.use_direct_dft = (on != 0)); }); }

int orc_set_variant(orc_ctx* c, double cs2, double f0, int kf, int evolve) {
    return guarded([&] {
        if (cs2 < 0 || kf < 0 || evolve < 0 || evolve > 3) throw std::invalid_argument("variant");
        DISPATCH(c, { S.cs2 = cs2; S.f0 = f0; S.kf = kf; S.evolve = evolve; S.have_old = false; });
    });
}
int orc_set_stress(orc_ctx* c, int on) {
    return guarded([&] { DISPATCH(c, { S.stress = on ? 1 : 0; S.have_old = false; }); });
}
int orc_set_integrator(orc_ctx* c, int integrator) {
    return guarded([&] {
        if (integrator < 0 || integrator > 2) throw std::invalid_argument("integrator");
        DISPATCH(c, { S.integrator = integrator; S.have_old = false; });
    });
}
int orc_set_fields(orc_ctx* c, int kind, const double* const f[8]) {
    return guarded([&] { if (kind != 0 && kind != 1) throw std::invalid_argument("kind"); DISPATCH(c, S.set_fields(kind, f)); });
}
int orc_get_fields(orc_ctx* c, int kind, double* const out[8]) {
    return guarded([&] { if (kind != 0 && kind != 1) throw std::invalid_argument("kind"); DISPATCH(c, S.get_fields(kind, out)); });
}
int orc_rhs(orc_ctx* c, double* const out[8]) { return guarded([&] { DISPATCH(c, rhs_out(S, out, nullptr, nullptr)); }); }
int orc_rhs_scales(orc_ctx* c, double* const out[8], double phi[8], double dsc[8]) {
    return guarded([&] { DISPATCH(c, rhs_out(S, out, phi, dsc)); });
}
int orc_step(orc_ctx* c, int nsteps) {
    return guarded([&] { DISPATCH(c, step_with_tracers(c, S, nsteps)); });
}
int orc_nspec(orc_ctx* c) { int n = 0; DISPATCH(c, n = S.nspec()); return n; }
int orc_diagnostics(orc_ctx* c, orc_diag* d, double* spec_kin, double* spec_mag, int nspec) {
    return guarded([&] {
        DISPATCH(c, {
            if (!S.have_fields) throw std::runtime_error("no fields set");
            if ((spec_kin || spec_mag) && nspec != S.nspec()) throw std::invalid_argument("nspec");
            orc::Diag g;
            S.diagnostics(g, spec_kin, spec_mag);
            d->t = g.t; d->step = g.step; d->ke = g.ke; d->me = g.me; d->ie = g.ie; d->mass = g.mass;
            for (int k = 0; k < 3; ++k) d->mom[k] = g.mom[k];
            d->etot = g.etot; d->max_divb = g.max_divb; d->rho_min = g.rho_min; d->p_min = g.p_min;
        });
    });
}
int orc_apply(orc_ctx* c, int op, const double* in, double* out) {
    return guarded([&] { if (op < 0 || op > 4) throw std::invalid_argument("op"); DISPATCH(c, apply_out(S, op, in, out)); });
}
int orc_fft3(int N, int sign, int precision, const double* in, double* out) {
    return guarded([&] { if (precision) transform<long double>(N, sign, false, in, out); else transform<double>(N, sign, false, in, out); });
}
int orc_dft3_direct(int N, int sign, int precision, const double* in, double* out) {
    return guarded([&] { if (precision) transform<long double>(N, sign, true, in, out); else transform<double>(N, sign, true, in, out); });
}

int orc_cic(int N, double L, int nf, const double* const g[], long long np, const double* const pos[3], double* const out[]) {
    return guarded([&] {
        if (N < 1 || !(L > 0) || nf < 1 || np < 0) throw std::invalid_argument("cic arguments");
        orc::tracers_interp(N, L, nf, g, np, pos, out);
    });
}
int orc_tracers_push(int N, double L, double dt, const double* const B[3], long long np, double* const pos[3],
                     double* const vel[3], int nsteps) {
    return guarded([&] {
        if (N < 1 || !(L > 0) || np < 0 || nsteps < 0) throw std::invalid_argument("push arguments");
        for (int s = 0; s < nsteps; ++s) orc::tracers_push(N, L, dt, B, np, pos, vel);
    });
}
int orc_tracers_set(orc_ctx* c, long long np, const double* const pos[3], const double* const vel[3]) {
    return guarded([&] {
        if (np < 0 || !pos) throw std::invalid_argument("tracers");
        c->np = np;
        for (int a = 0; a < 3; ++a) {
            c->tpos[a].assign(pos[a], pos[a] + np);
            c->tvel[a].assign(np, 0.0);
        }
        DISPATCH(c, tracers_attach(c, S, np, vel));
    });
}
int orc_tracers_get(orc_ctx* c, double* const pos[3], double* const vel[3]) {
    return guarded([&] {
        for (int a = 0; a < 3; ++a) {
            if (pos) std::copy(c->tpos[a].begin(), c->tpos[a].end(), pos[a]);
            if (vel) std::copy(c->tvel[a].begin(), c->tvel[a].end(), vel[a]);
        }
    });
}

}  // extern "C"

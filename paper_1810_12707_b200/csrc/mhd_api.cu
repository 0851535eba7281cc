// mhd_api.cu — context, workspace layout, sweep orchestration and the C ABI of include/mhd.h.
//
// State lives in k-space: U^ (8 half-spectrum arrays, zero outside the 2/3 mask) and the Adams-Bashforth history
// R^old.  One right-hand side is five sweeps over HBM:
//   S1  build J^ = i k x B^ ; inverse z pass of (U^, J^) -> W[0..10]          (pruned: only modes inside the mask)
//   S2  inverse y pass, in place
//   S3  x_fused: C2R of 11 fields, flux products, R2C of 16 products, in place on W[0..15]
//   S4  forward y pass, in place
//   S5  forward z pass ; assembly of R^ (i k, -k^2, mask) and the explicit update
// No host round trip inside mhd_step: only kernel launches on the bound stream.
#include "ctx.h"

#include <mutex>
#include <set>
#include <utility>

using namespace mhd;

namespace mhd {
namespace { thread_local std::string t_config_error; }
cudaError_t configure_kernel(const void* kern, size_t smem, bool nonportable_cluster) {
    static std::mutex mu;
    static std::set<std::pair<const void*, int>> done;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(mu);          // held across the set: nobody sees (kern, dev) before it is configured
    const auto key = std::make_pair(kern, dev);
    if (done.count(key)) return cudaSuccess;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    // clusters of 16 are above the portable size of 8: a per-function, per-device opt-in
    if (e == cudaSuccess && nonportable_cluster) e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    if (e != cudaSuccess) {
        t_config_error = std::string("cudaFuncSetAttribute (") + std::to_string(smem) + " B of dynamic shared memory" +
                         (nonportable_cluster ? ", non-portable cluster size" : "") + "): " + cudaGetErrorString(e);
        return e;                                  // not recorded: the next launch tries again
    }
    done.insert(key);
    return cudaSuccess;
}
const char* kernel_config_error() {
    static thread_local std::string out;
    out.swap(t_config_error);
    t_config_error.clear();
    return out.c_str();
}
}  // namespace mhd

namespace {

// ---- sweeps --------------------------------------------------------------------------------------------------
// strided pass over nf arrays; axis 1 = y, 2 = z; hx = row pitch of the arrays (N/2, or 8 for the Nyquist planes)
// axis 1 only: z0 / nz restrict the pass to the z planes [z0, z0 + nz) (nz = 0: all planes) — the L2 slab loop
void strided_pass(mhd_ctx* c, int dir, int axis, int nf, const cd* const in[], cd* const out[], int hx, int ncols_full,
                  bool prune, int jfirst = -1, int bfirst = 0, int z0 = 0, int nz = 0) {
    const int N = c->N, kc = c->kc();
    int done = 0;
    while (done < nf) {
        const int nb = std::min(nf - done, MAXF);
        StridedArgs a;
        std::memset(&a, 0, sizeof(a));
        const long long zoff = (axis == 1 && nz > 0) ? (long long)z0 * N * hx : 0;
        for (int f = 0; f < nb; ++f) { a.in[f] = in[done + f] + zoff; a.out[f] = out[done + f] + zoff; }
        a.tw = c->tw;
        a.kc = kc;
        a.nfields = nb;
        a.jfirst = jfirst; a.bfirst = bfirst; a.k0 = 2.0 * M_PI / c->L;   // fused current: only with nf <= MAXF
        a.ncols = prune ? std::min(kc + 1, ncols_full) : ncols_full;
        if (axis == 1) {            // y pass: rows along y, outer = z (all planes)
            a.in_row_stride = a.out_row_stride = hx; a.in_outer_stride = a.out_outer_stride = (long long)N * hx;
            a.n_outer = nz > 0 ? nz : N; a.outer_split = N; a.outer_skip = 0;
        } else {                    // z pass: rows along z, outer = ky (pruned to the mask)
            a.in_row_stride = a.out_row_stride = (long long)N * hx; a.in_outer_stride = a.out_outer_stride = hx;
            if (prune) { a.n_outer = 2 * kc + 1; a.outer_split = kc + 1; a.outer_skip = N - (2 * kc + 1); }
            else { a.n_outer = N; a.outer_split = N; a.outer_skip = 0; }
        }
        a.in_rows = (prune && dir > 0) ? 1 : 0;     // inverse: input rows outside the mask are zero
        a.out_rows = (prune && dir < 0) ? 1 : 0;    // forward: output rows outside the mask are not needed
        mhd_ctx::Scope s(c, dir > 0 ? F_STRIDED_INV : F_STRIDED_FWD);
        const bool tma = c->opt_tma != 0 && zoff == 0;      // MHD_OPT_TMA (opt-in: measured slower than the register-fed kernel)
        if (tma && launch_strided_tma(N, dir, a, c->tma, c->st)) ++c->tma_launches;
        else launch_strided(N, dir, a, c->st);
        done += nb;
    }
}

// spec (destroyed unless work != spec) -> real.  work may alias spec; real_out may alias work.
void inverse3d(mhd_ctx* c, int nf, const cd* const spec[], cd* const work[], double* const real_out[], bool prune) {
    const int N = c->N;
    strided_pass(c, +1, 2, nf, spec, work, c->hx(), c->hx(), prune);
    strided_pass(c, +1, 1, nf, work, work, c->hx(), c->hx(), prune);
    int done = 0;
    while (done < nf) {
        const int nb = std::min(nf - done, MAXF);
        XArgs a; std::memset(&a, 0, sizeof(a));
        for (int f = 0; f < nb; ++f) { a.spec_in[f] = work[done + f]; a.real_out[f] = real_out[done + f]; }
        a.tw = c->tw; a.nlines = (long long)N * N; a.nfields = nb;
        a.kmax = prune ? c->kc() : c->hx() - 1;
        a.scale = 1.0 / ((double)N * N * N);
        mhd_ctx::Scope s(c, F_X_C2R);
        launch_x_c2r(N, a, c->st);
        done += nb;
    }
}

// real -> spec (may alias real storage); nyq (optional, unpruned only) receives the kx = N/2 plane
void forward3d(mhd_ctx* c, int nf, const double* const real_in[], cd* const spec[], cd* const nyq[], bool prune) {
    const int N = c->N;
    int done = 0;
    while (done < nf) {
        const int nb = std::min(nf - done, MAXF);
        XArgs a; std::memset(&a, 0, sizeof(a));
        for (int f = 0; f < nb; ++f) {
            a.real_in[f] = real_in[done + f]; a.spec_out[f] = spec[done + f];
            a.nyq_out[f] = nyq ? nyq[done + f] : nullptr;
        }
        a.tw = c->tw; a.nlines = (long long)N * N; a.nfields = nb;
        a.kmax = prune ? c->kc() : c->hx() - 1;
        a.scale = 1.0;
        mhd_ctx::Scope s(c, F_X_R2C);
        launch_x_r2c(N, a, c->st);
        done += nb;
    }
    strided_pass(c, -1, 1, nf, spec, spec, c->hx(), c->hx(), prune);
    strided_pass(c, -1, 2, nf, spec, spec, c->hx(), c->hx(), prune);
    if (nyq) {
        strided_pass(c, -1, 1, nf, nyq, nyq, 8, 1, false);
        strided_pass(c, -1, 2, nf, nyq, nyq, 8, 1, false);
    }
}

}  // namespace

void run_x_fused(mhd_ctx* c, cd* const in[11], cd* const out[16], long long nlines, double* const breal[3]) {
    const int N = c->N;
    const bool prune = c->opt_prune != 0 || c->ooc.on;
    const int kmax = prune ? c->kc() : c->hx() - 1;
    FusedXArgs a; std::memset(&a, 0, sizeof(a));
    for (int f = 0; f < 11; ++f) a.in[f] = in[f];
    for (int f = 0; f < 16; ++f) a.out[f] = out[f];
    a.tw = c->tw; a.nlines = nlines; a.kmax_in = kmax; a.kmax_out = kmax;
    a.scale = 1.0 / ((double)N * N * N); a.ph = c->phys();
    const bool gen2 = c->opt_fused != 2 && x_fused2_supported(N);
    if (breal && gen2) for (int d = 0; d < 3; ++d) a.breal[d] = breal[d];   // only the second-generation kernel emits B
    mhd_ctx::Scope s(c, F_X_FUSED);
    if (gen2) { a.tw = c->ftw; launch_x_fused2(N, a, c->st); }
    else launch_x_fused(N, a, c->st);
}

namespace {

// products W[0..15] <- state Uin (k-space); sweeps S1-S4 and the forward z pass of S5
// breal != null (tracers, fused sweep only): the real-space B of Uin is also written there by sweep S3
// s5a = false: the forward z pass is left to the caller (fused with the assembly: sweep S5 in one launch)
void products(mhd_ctx* c, cd* const Uin[8], double* const breal[3] = nullptr, bool s5a = true) {
    const int N = c->N;
    const bool prune = c->opt_prune != 0;
    const SpecGeom g = c->geom();
    const Phys ph = c->phys();
    const cd* in[11];
    for (int f = 0; f < 8; ++f) in[f] = Uin[f];
    for (int f = 8; f < 11; ++f) in[f] = c->W[f];
    if (c->opt_fused && c->opt_fuse_current) {
        // S1: inverse z pass of U^ with J^ = M i k x B^ built on load (fields 8..10 come from in[5..7])
        strided_pass(c, +1, 2, 11, in, c->W, c->hx(), c->hx(), prune, 8, 5);
    } else {
        {   // S1a: J^ = M i k x B^ -> W[8..10]
            mhd_ctx::Scope s(c, F_CURRENT);
            launch_build_current(g, Uin + 5, c->W + 8, ph, c->st);
        }
        strided_pass(c, +1, 2, 11, in, c->W, c->hx(), c->hx(), prune);    // S1b
    }
    // S2-S4 work inside z planes; one launch per sweep over the whole volume (a slab-after-slab loop that keeps the
    // intermediates in L2 measured slower at every slab size: DESIGN.md "L2 slab loop")
    const int kmax = prune ? c->kc() : c->hx() - 1;
    const double scale = 1.0 / ((double)N * N * N);
    const int slab = N;
    for (int z0 = 0; z0 < N; z0 += slab) {
        const int nz = std::min(slab, N - z0);
        strided_pass(c, +1, 1, 11, c->W, c->W, c->hx(), c->hx(), prune, -1, 0, z0, nz);      // S2
        if (c->opt_fused) {                                                                 // S3
            const long long off = (long long)z0 * N * c->hx();
            cd* w[16];
            for (int f = 0; f < 16; ++f) w[f] = c->W[f] + off;
            double* br[3] = {nullptr, nullptr, nullptr};
            if (breal) for (int d = 0; d < 3; ++d) br[d] = breal[d] + 2 * off;
            run_x_fused(c, w, w, (long long)nz * N, breal ? br : nullptr);
        } else {
            XArgs a; std::memset(&a, 0, sizeof(a));
            for (int f = 0; f < 11; ++f) { a.spec_in[f] = c->W[f]; a.real_out[f] = reinterpret_cast<double*>(c->W[f]); }
            a.tw = c->tw; a.nlines = (long long)N * N; a.nfields = 11; a.kmax = kmax; a.scale = scale;
            { mhd_ctx::Scope s(c, F_X_C2R); launch_x_c2r(N, a, c->st); }
            const double* rin[11]; double* rout[16];
            for (int f = 0; f < 11; ++f) rin[f] = reinterpret_cast<const double*>(c->W[f]);
            for (int f = 0; f < 16; ++f) rout[f] = reinterpret_cast<double*>(c->W[f]);
            { mhd_ctx::Scope s(c, F_FLUX); launch_flux_real(c->n3(), rin, rout, ph, c->st); }
            XArgs b; std::memset(&b, 0, sizeof(b));
            for (int f = 0; f < 16; ++f) { b.real_in[f] = rout[f]; b.spec_out[f] = c->W[f]; }
            b.tw = c->tw; b.nlines = (long long)N * N; b.nfields = 16; b.kmax = kmax; b.scale = 1.0;
            { mhd_ctx::Scope s(c, F_X_R2C); launch_x_r2c(N, b, c->st); }
        }
        strided_pass(c, -1, 1, 16, c->W, c->W, c->hx(), c->hx(), prune, -1, 0, z0, nz);      // S4
    }
    if (s5a) strided_pass(c, -1, 2, 16, c->W, c->W, c->hx(), c->hx(), prune);      // S5a
}

// sweep S5 in one launch: forward z pass of W[0..15] + assembly + update (kernels.h AssembleTail)
StridedArgs s5_args(mhd_ctx* c) {
    const int N = c->N, kc = c->kc(), hx = c->hx();
    StridedArgs a;
    std::memset(&a, 0, sizeof(a));
    for (int f = 0; f < 16; ++f) { a.in[f] = c->W[f]; a.out[f] = c->W[f]; }
    a.tw = c->tw; a.kc = kc; a.nfields = 16; a.jfirst = -1;
    a.ncols = std::min(kc + 1, hx);
    a.in_row_stride = a.out_row_stride = (long long)N * hx; a.in_outer_stride = a.out_outer_stride = hx;
    a.n_outer = 2 * kc + 1; a.outer_split = kc + 1; a.outer_skip = N - (2 * kc + 1);
    a.in_rows = 0; a.out_rows = 1;
    return a;
}
// can this device co-schedule the kernel's thread-block clusters (16 CTAs are above the portable size)?  Asked once per
// context and variant; "no" makes rhs_spectral keep the two-launch sweep instead of failing the step at launch time
bool s5_available(mhd_ctx* c) {
    const int v = c->opt_fuse_assemble;
    if (v < 1 || v > 2 || !strided_assemble_supported(c->N)) return false;
    if (c->s5_ok[v] < 0) {
        c->s5_ok[v] = strided_assemble_max_clusters(c->N, v, s5_args(c)) > 0 ? 1 : 0;
        cudaGetLastError();                 // an unavailable cluster shape is an answer, not an error of the step
        kernel_config_error();
    }
    return c->s5_ok[v] == 1;
}
void fused_s5(mhd_ctx* c, cd* const Uin[8], cd* const rout[8], int mode) {
    const StridedArgs a = s5_args(c);
    AssembleTail z;
    std::memset(&z, 0, sizeof(z));
    for (int f = 0; f < 8; ++f) { z.U[f] = Uin[f]; z.Rold[f] = c->Rold[f]; z.rout[f] = rout ? rout[f] : nullptr; }
    z.mode = mode; z.dt = c->dt; z.ph = c->phys();
    mhd_ctx::Scope s(c, F_S5);
    launch_strided_assemble(c->N, c->opt_fuse_assemble, a, z, c->st);
    ++c->s5_launches;
}

// Variant MHD_OPT_STRESS (Eq. 3-4, 11-12): V_ij = 2 nu rho S_ij and Wv_j = u_i V_ij, transformed, for the assembly.
// An unfused add-on pass (22 extra 3-D transforms): Uin -> real rho, m -> u = m/rho -> u^ -> S^ -> real S -> V, Wv -> V^, Wv^.
// Buffers: X[0..3] real rho, m; X[4..6] real u; u^ in Y[6], Y[7], X[7]; S / V in Y[0..5]; Wv over u^.
void viscous_pass(mhd_ctx* c, cd* const Uin[8]) {
    const long long n3 = c->n3();
    SpecGeom gp = c->geom(); gp.pruned = 1;
    const cd* spec4[4] = {Uin[0], Uin[1], Uin[2], Uin[3]};
    cd* work4[4] = {c->X[0], c->X[1], c->X[2], c->X[3]};
    double* real4[4];
    for (int f = 0; f < 4; ++f) real4[f] = reinterpret_cast<double*>(c->X[f]);
    inverse3d(c, 4, spec4, work4, real4, true);
    double* u[3] = {reinterpret_cast<double*>(c->X[4]), reinterpret_cast<double*>(c->X[5]), reinterpret_cast<double*>(c->X[6])};
    const double* m[3] = {real4[1], real4[2], real4[3]};
    { mhd_ctx::Scope s(c, F_POINT); launch_velocity_real(n3, real4[0], m, u, c->st); }
    const double* uc[3] = {u[0], u[1], u[2]};
    cd* uhat[3] = {c->Y[6], c->Y[7], c->X[7]};
    forward3d(c, 3, uc, uhat, nullptr, true);
    const cd* uhc[3] = {uhat[0], uhat[1], uhat[2]};
    cd* S[6] = {c->Y[0], c->Y[1], c->Y[2], c->Y[3], c->Y[4], c->Y[5]};
    { mhd_ctx::Scope s(c, F_POINT); launch_strain_spec(gp, uhc, S, c->phys(), c->st); }
    const cd* Sc[6]; double* Sr[6];
    for (int f = 0; f < 6; ++f) { Sc[f] = S[f]; Sr[f] = reinterpret_cast<double*>(S[f]); }
    inverse3d(c, 6, Sc, S, Sr, true);
    double* Wv[3] = {reinterpret_cast<double*>(uhat[0]), reinterpret_cast<double*>(uhat[1]), reinterpret_cast<double*>(uhat[2])};
    { mhd_ctx::Scope s(c, F_POINT); launch_viscous_flux(n3, c->mu, real4[0], uc, Sr, Wv, c->st); }
    const double* r9[9]; cd* s9[9];
    for (int f = 0; f < 6; ++f) { r9[f] = Sr[f]; s9[f] = S[f]; }
    for (int f = 0; f < 3; ++f) { r9[6 + f] = Wv[f]; s9[6 + f] = uhat[f]; }
    forward3d(c, 9, r9, s9, nullptr, true);
}

// R^(Uin) -> rout (mode 0) or explicit update of Uin / Rold (mode 1 Euler, 2 AB2)
void rhs_spectral(mhd_ctx* c, cd* const Uin[8], cd* const rout[8], int mode, double* const breal[3] = nullptr,
                  const StageUpdate* stage = nullptr) {
    const bool stress = c->opt_stress != 0;
    const cd* visc[9] = {c->Y[0], c->Y[1], c->Y[2], c->Y[3], c->Y[4], c->Y[5], c->Y[6], c->Y[7], c->X[7]};
    if (stress) viscous_pass(c, Uin);                 // V^_ij, Wv^_j -> Y[0..7], X[7]   (before the products: uses X, Y)
    const bool forced = c->f0 != 0.0;
    // default equation set on the pruned, fused path: sweep S5 is one launch
    const bool one_s5 = c->opt_fuse_assemble != 0 && c->opt_fused != 0 && c->opt_prune != 0 && !stress && !forced &&
                        c->cs2 <= 0.0 && c->evolve == 3 && mode != 3 && s5_available(c);
    products(c, Uin, breal, !one_s5);
    if (one_s5) { fused_s5(c, Uin, rout, mode); return; }
    SpecGeom gp = c->geom(); gp.pruned = 1;
    const cd* Uc[8];
    for (int f = 0; f < 8; ++f) Uc[f] = Uin[f];
    cd* fbuf[4] = {c->X[3], c->X[4], c->X[5], c->X[6]};           // X[0..2] may hold the tracers' real-space B
    const cd* force[4] = {fbuf[0], fbuf[1], fbuf[2], fbuf[3]};
    if (forced && mode != 0) {      // the update is in place: the +-k_f neighbours of U^ must be read before it starts
        mhd_ctx::Scope s(c, F_POINT);
        launch_forcing(gp, Uc, fbuf, 0, c->phys(), c->st);
    }
    {
        Phys ph = c->phys();
        if (stress) ph.mu = 0.0;                      // the viscous terms come from `visc`, not from mu k^2 u^
        mhd_ctx::Scope s(c, F_ASSEMBLE);
        launch_assemble(c->geom(), c->W, Uin, c->Rold, rout, mode, c->dt, ph, c->st, (forced && mode != 0) ? force : nullptr,
                        stress ? visc : nullptr, stage);
    }
    if (forced && mode == 0) {      // U^ is not modified: add F^ to the assembled R^ (X, Y may hold integrator stages)
        mhd_ctx::Scope s(c, F_POINT);
        launch_forcing(gp, Uc, rout, 1, c->phys(), c->st);
    }
}

// ---- tracer particles (Sec. VI) ----------------------------------------------------------------------
TracerArgs tracer_args(mhd_ctx* c, const double* const B[3], int nsteps) {
    TracerArgs a; std::memset(&a, 0, sizeof(a));
    for (int d = 0; d < 3; ++d) { a.B[d] = B ? B[d] : nullptr; a.pos[d] = c->tr.pos[d]; a.vel[d] = c->tr.vel[d]; }
    a.np = c->tr.np; a.N = c->N; a.L = c->L; a.dt = c->dt; a.nsteps = nsteps;
    return a;
}
bool tracers_active(const mhd_ctx* c) { return c->tr.np > 0 && c->tr.set; }
// sweep S3 of the second-generation fused kernel can write the real-space B as a by-product
bool tracers_fused_emit(const mhd_ctx* c) { return c->opt_fused == 1 && x_fused2_supported(c->N) && c->integrator == 0; }
// real-space B of the current state -> X[0..2] by a separate pruned inverse transform (U^ is left intact).
// Returns MHD_OK or the error of the chunked slab stage (staging overflow, decomposed context, ...): the caller must not
// push particles in a B that was never written.
int tracers_real_B(mhd_ctx* c, double* Breal[3]) {
    if (c->ooc.on) {            // chunked pipeline: the slab stage of mhd_get_fields, B only, into the tracers' own arrays
        double* out[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, c->tr.field[0], c->tr.field[1], c->tr.field[2]};
        for (int d = 0; d < 3; ++d) Breal[d] = c->tr.field[d];
        return ooc_real_fields(c, out);
    }
    const cd* spec[3] = {c->U[5], c->U[6], c->U[7]};
    cd* work[3] = {c->X[0], c->X[1], c->X[2]};
    for (int d = 0; d < 3; ++d) Breal[d] = reinterpret_cast<double*>(c->X[d]);
    inverse3d(c, 3, spec, work, Breal, true);
    return MHD_OK;
}
// spatial sort of the particle storage (tracers.cu); ping-pongs the two sets of arrays
void tracers_sort(mhd_ctx* c) {
    auto& t = c->tr;
    {
        mhd_ctx::Scope s(c, F_TRACERS, 3);
        launch_tracer_sort(tracer_args(c, nullptr, 0), t.id, t.alt, t.alt_id, t.hist, t.key, t.rank, c->st);
    }
    for (int d = 0; d < 3; ++d) { std::swap(t.pos[d], t.alt[d]); std::swap(t.vel[d], t.alt[3 + d]); }
    std::swap(t.id, t.alt_id);
    t.sorted = true; t.since_sort = 0;
}
// nsteps pushes in the field Breal; the storage is re-sorted every opt_tracer_sort pushes
void tracers_push_with(mhd_ctx* c, double* const Breal[3], int nsteps) {
    const double* B[3] = {Breal[0], Breal[1], Breal[2]};
    const int every = c->opt_tracer_sort;
    while (nsteps > 0) {
        if (every > 0 && c->tr.since_sort >= every) tracers_sort(c);
        const int n = every > 0 ? std::min(nsteps, every - c->tr.since_sort) : nsteps;
        mhd_ctx::Scope s(c, F_TRACERS);
        launch_tracer_push(tracer_args(c, B, n), c->st);
        c->tr.since_sort += n; nsteps -= n;
    }
}

int copy_in(mhd_ctx* c, int where, const double* const src[8], double* const dst[8]) {
    const size_t bytes = (size_t)c->n3() * sizeof(double);
    for (int f = 0; f < 8; ++f) {
        if (!src[f]) return c->fail(MHD_ERR_INVALID_ARG, "null field pointer");
        cudaMemcpyAsync(dst[f], src[f], bytes, where == MHD_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, c->st);
    }
    return check_cuda(c, "copy in");
}
int copy_out(mhd_ctx* c, int where, double* const src[8], double* const dst[8]) {
    const size_t bytes = (size_t)c->n3() * sizeof(double);
    for (int f = 0; f < 8; ++f) {
        if (!dst[f]) return c->fail(MHD_ERR_INVALID_ARG, "null field pointer");
        if (dst[f] != src[f])
            cudaMemcpyAsync(dst[f], src[f], bytes, where == MHD_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, c->st);
    }
    if (where == MHD_HOST) cudaStreamSynchronize(c->st);
    return check_cuda(c, "copy out");
}

}  // namespace

// =====================================================================================================================
extern "C" {

int mhd_init(mhd_ctx** out, int N, double L, double gamma, double mu, double eta, double dt) {
    if (!out) return MHD_ERR_INVALID_ARG;
    *out = nullptr;
    if (!valid_N(N) || !(L > 0) || !(gamma > 1) || !(mu >= 0) || !(eta >= 0) || !(dt > 0)) return MHD_ERR_INVALID_ARG;
    mhd_ctx* c = new (std::nothrow) mhd_ctx();
    if (!c) return MHD_ERR_NOMEM;
    c->N = N; c->L = L; c->gamma = gamma; c->mu = mu; c->eta = eta; c->dt = dt;
    *out = c;
    return MHD_OK;
}

static bool flags_valid(unsigned flags) {
    if ((flags & 0x80u) != 0) return false;                                 // unknown bits
    if ((flags & 0x70u) && (flags & (MHD_FLAG_STATE_ON_HOST | MHD_FLAG_WORK_ON_HOST))) return false;   // per-rank storage lives in HBM
    if (!(flags & MHD_FLAG_OUT_OF_CORE)) return flags == 0;                 // placement / budget need the chunked pipeline
    return true;
}
size_t mhd_workspace_bytes(int N, unsigned flags) {
    if (!valid_N(N) || !flags_valid(flags)) return 0;
    if (flags & MHD_FLAG_OUT_OF_CORE) return ooc_workspace_bytes(N, flags);
    return make_layout(N).total;
}
size_t mhd_pinned_bytes(int N, unsigned flags) {
    if (!valid_N(N) || !flags_valid(flags) || !(flags & MHD_FLAG_OUT_OF_CORE)) return 0;
    return ooc_pinned_bytes(N, flags);
}
int mhd_nspec(int N) { return nspec_of(N); }

int mhd_bind(mhd_ctx* c, void* dev_workspace, size_t bytes, void* cuda_stream, unsigned flags, void* pinned_host,
             size_t pinned_bytes) {
    if (!c) return MHD_ERR_INVALID_ARG;
    if (!flags_valid(flags)) return c->fail(MHD_ERR_INVALID_ARG, "invalid flags");
    if ((flags & MHD_FLAG_OUT_OF_CORE) && (c->f0 != 0.0 || c->opt_stress))     // set before binding: refuse here, not silently later
        return c->fail(MHD_ERR_INVALID_ARG, "forcing / the stress-tensor variant were set: they need an in-core context");
    if (!dev_workspace || ((uintptr_t)dev_workspace & 255) != 0) return c->fail(MHD_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
    const Layout l = make_layout(c->N);
    if (!(flags & MHD_FLAG_OUT_OF_CORE) && bytes < l.total) return c->fail(MHD_ERR_NOMEM, "workspace too small");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return c->fail(MHD_ERR_CUDA, "no CUDA device (libmhd has no CPU fallback)");
    }
    char* base = static_cast<char*>(dev_workspace);
    c->st = static_cast<cudaStream_t>(cuda_stream);
    c->flags = flags;
    if (flags & MHD_FLAG_OUT_OF_CORE) {
        int rc = ooc_bind(c, base, bytes, static_cast<char*>(pinned_host), pinned_bytes);
        if (rc) return rc;
        c->bound = true; c->have_fields = false; c->have_old = false; c->step = 0;
        return MHD_OK;
    }
    c->ooc.on = false;
    c->tw = reinterpret_cast<cd*>(base + l.tw_off);
    c->ftw = reinterpret_cast<cd*>(base + l.ftw_off);
    const size_t fb = align_up(l.field_bytes);
    char* fp = base + l.field_off;
    int k = 0;
    for (int f = 0; f < 8; ++f) c->U[f] = reinterpret_cast<cd*>(fp + (size_t)(k++) * fb);
    for (int f = 0; f < 8; ++f) c->Rold[f] = reinterpret_cast<cd*>(fp + (size_t)(k++) * fb);
    for (int f = 0; f < 16; ++f) c->W[f] = reinterpret_cast<cd*>(fp + (size_t)(k++) * fb);
    for (int f = 0; f < 8; ++f) c->X[f] = reinterpret_cast<cd*>(fp + (size_t)(k++) * fb);
    for (int f = 0; f < 8; ++f) c->Y[f] = reinterpret_cast<cd*>(fp + (size_t)(k++) * fb);
    for (int f = 0; f < 3; ++f) c->nyq[f] = reinterpret_cast<cd*>(base + l.nyq_off + (size_t)f * l.nyq_bytes);
    c->scratch = reinterpret_cast<double*>(base + l.scratch_off);
    c->res = reinterpret_cast<double*>(base + l.res_off);
    launch_twiddle_table(c->N, c->tw, c->st);
    launch_x_fused2_tables(c->N, c->ftw, c->st);
    c->launches += 2;
    c->tma = StridedTma();
    if (strided_tma_supported(c->N) && strided_tma_build_maps(c->N, fp, fb, NFIELD_BUFS, c->tmaps)) {
        int dev = 0, sms = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        c->tma.maps = c->tmaps; c->tma.base = fp; c->tma.stride_bytes = fb; c->tma.nbuf = NFIELD_BUFS; c->tma.sms = sms;
    }
    int rc = check_cuda(c, "bind");
    if (rc) return rc;
    c->bound = true; c->have_fields = false; c->have_old = false; c->step = 0;
    return MHD_OK;
}

int mhd_set_option(mhd_ctx* c, int option, int value) {
    if (!c) return MHD_ERR_INVALID_ARG;
    switch (option) {
        case MHD_OPT_FUSED:
            if (value < 0 || value > 2) return c->fail(MHD_ERR_INVALID_ARG, "fused must be 0, 1 or 2");
            c->opt_fused = value; return MHD_OK;
        case MHD_OPT_PRUNE: c->opt_prune = value ? 1 : 0; return MHD_OK;
        case MHD_OPT_FUSE_CURRENT: c->opt_fuse_current = value ? 1 : 0; return MHD_OK;
        case MHD_OPT_TMA:
            // a bound context knows whether its tensor maps could be built: refuse instead of silently running the default
            if (value && c->bound && !c->ooc.on && !c->tma.maps)
                return c->fail(MHD_ERR_INVALID_ARG, "the TMA pipeline is not available for this context (N must be 128, 256 or 512 and "
                                                    "cuTensorMapEncodeTiled must succeed)");
            c->opt_tma = value ? 1 : 0; return MHD_OK;
        case 7: case 10:
            return c->fail(MHD_ERR_INVALID_ARG, "option ids 7 and 10 are retired (include/mhd_bench.h)");
        case MHD_OPT_FUSE_ASSEMBLE:
            if (value < 0 || value > 2) return c->fail(MHD_ERR_INVALID_ARG, "fuse_assemble must be 0, 1 or 2");
            c->opt_fuse_assemble = value; return MHD_OK;
        case MHD_OPT_INTEGRATOR:
            if (value < 0 || value > 2) return c->fail(MHD_ERR_INVALID_ARG, "integrator must be 0, 1 or 2");
            c->integrator = value; c->have_old = false; return MHD_OK;
        case MHD_OPT_TRACER_SORT:
            if (value < 0) return c->fail(MHD_ERR_INVALID_ARG, "tracer sort interval must be >= 0");
            c->opt_tracer_sort = value; return MHD_OK;
        case MHD_OPT_STRESS:
            if (value != 0 && c->ooc.on) return c->fail(MHD_ERR_INVALID_ARG, "the stress-tensor variant needs an in-core context");
            c->opt_stress = value ? 1 : 0; c->have_old = false; return MHD_OK;
        case MHD_OPT_EVOLVE:
            if (value < 0 || value > 3) return c->fail(MHD_ERR_INVALID_ARG, "evolve must be 0..3");
            c->evolve = value; c->have_old = false; return MHD_OK;
        case MHD_OPT_FORCE_K:
            if (value < 1 || value > c->kc()) return c->fail(MHD_ERR_INVALID_ARG, "forcing mode must be in 1..kc");
            c->kf = value; c->have_old = false; return MHD_OK;
        case MHD_OPT_OOC_BRICK:
            if (value < 0) return c->fail(MHD_ERR_INVALID_ARG, "brick size must be >= 0");
            c->ooc.brick_max = value; return MHD_OK;
        case MHD_OPT_OOC_SLAB:
            if (value < 0) return c->fail(MHD_ERR_INVALID_ARG, "slab size must be >= 0");
            c->ooc.slab_max = value; return MHD_OK;
        default: return c->fail(MHD_ERR_INVALID_ARG, "unknown option");
    }
}

long long mhd_alt_launch_count(const mhd_ctx* c, int which) {
    if (!c) return -1;
    if (which == MHD_OPT_TMA) return c->tma_launches;
    if (which == MHD_OPT_FUSE_ASSEMBLE) return c->s5_launches;
    return -1;
}

int mhd_set_param(mhd_ctx* c, int param, double value) {
    if (!c) return MHD_ERR_INVALID_ARG;
    switch (param) {
        case MHD_PARAM_CS2:
            if (!(value >= 0.0)) return c->fail(MHD_ERR_INVALID_ARG, "C_s^2 must be >= 0");
            c->cs2 = value; c->have_old = false; return MHD_OK;
        case MHD_PARAM_FORCE_AMP:
            if (value != value) return c->fail(MHD_ERR_INVALID_ARG, "forcing amplitude is NaN");
            if (value != 0.0 && c->ooc.on) return c->fail(MHD_ERR_INVALID_ARG, "forcing needs an in-core context");
            c->f0 = value; c->have_old = false; return MHD_OK;
        default: return c->fail(MHD_ERR_INVALID_ARG, "unknown parameter");
    }
}

int mhd_set_fields(mhd_ctx* c, int kind, int where, const double* const f[8]) {
    if (!c || !f) return MHD_ERR_INVALID_ARG;
    if (!c->bound) return c->fail(MHD_ERR_NOT_BOUND, "mhd_bind has not been called");
    if ((kind != 0 && kind != 1) || (where != 0 && where != 1)) return c->fail(MHD_ERR_INVALID_ARG, "kind/where");
    if (c->ooc.on) {
        int rc = ooc_set_fields(c, kind, where, f);
        if (rc) return rc;
        c->have_fields = c->ooc.world == 1;      // decomposed: only after the exchange and MHD_DIST_PHASE_STORE
        c->have_old = false; c->step = 0;
        return MHD_OK;
    }
    double* real[8];
    for (int i = 0; i < 8; ++i) real[i] = reinterpret_cast<double*>(c->W[i]);
    int rc = copy_in(c, where, f, real);
    if (rc) return rc;
    if (kind == MHD_PRIMITIVE) { mhd_ctx::Scope s(c, F_POINT); launch_prim_to_cons(c->n3(), real, c->gamma, c->st); }
    const size_t bytes = (size_t)c->n3() * sizeof(double);
    for (int i = 0; i < 8; ++i) cudaMemsetAsync(c->U[i], 0, bytes, c->st);
    // projection U <- M FFT U: the pruned forward transform writes exactly the modes inside the mask
    const double* rin[8];
    for (int i = 0; i < 8; ++i) rin[i] = real[i];
    forward3d(c, 8, rin, c->W, nullptr, true);
    {
        SpecGeom g = c->geom(); g.pruned = 1;
        const cd* src[8];
        for (int i = 0; i < 8; ++i) src[i] = c->W[i];
        mhd_ctx::Scope s(c, F_AXPBY);
        launch_copy_masked(g, 8, c->U, src, c->st);
    }
    if (where == MHD_HOST) cudaStreamSynchronize(c->st);
    rc = check_cuda(c, "set_fields");
    if (rc) return rc;
    c->have_fields = true; c->have_old = false; c->step = 0;
    return MHD_OK;
}

int mhd_rhs(mhd_ctx* c, int where, double* const out[8]) {
    if (!c || !out) return MHD_ERR_INVALID_ARG;
    if (!c->bound) return c->fail(MHD_ERR_NOT_BOUND, "mhd_bind has not been called");
    if (!c->have_fields) return c->fail(MHD_ERR_NO_FIELDS, "mhd_set_fields has not been called");
    if (where != 0 && where != 1) return c->fail(MHD_ERR_INVALID_ARG, "where");
    if (c->ooc.on) return ooc_rhs(c, where, out);
    rhs_spectral(c, c->U, c->X, 0);
    double* real[8];
    for (int i = 0; i < 8; ++i) real[i] = (where == MHD_DEVICE) ? out[i] : reinterpret_cast<double*>(c->X[i]);
    inverse3d(c, 8, c->X, c->X, real, c->opt_prune != 0);
    int rc = copy_out(c, where, real, out);
    return rc ? rc : check_cuda(c, "rhs");
}

int mhd_step(mhd_ctx* c, int nsteps) {
    if (!c || nsteps < 0) return MHD_ERR_INVALID_ARG;
    if (!c->bound) return c->fail(MHD_ERR_NOT_BOUND, "mhd_bind has not been called");
    if (!c->have_fields) return c->fail(MHD_ERR_NO_FIELDS, "mhd_set_fields has not been called");
    if (c->ooc.on) {
        if (!tracers_active(c)) return ooc_step(c, nsteps);
        for (int s = 0; s < nsteps; ++s) {      // tracers feel the B of the state at the start of each step
            double* Breal[3];
            if (int rc = tracers_real_B(c, Breal)) return rc;
            tracers_push_with(c, Breal, 1);
            if (int rc = ooc_step(c, 1)) return rc;
        }
        return check_cuda(c, "step (chunked, tracers)");
    }
    const SpecGeom g = c->geom();
    SpecGeom gp = g; gp.pruned = 1;
    if (c->opt_stress && c->integrator != 0) return c->fail(MHD_ERR_INVALID_ARG, "the stress-tensor variant is implemented for Adams-Bashforth only");
    const bool tracers = tracers_active(c), emit = tracers && tracers_fused_emit(c);
    double* Breal[3] = {reinterpret_cast<double*>(c->X[0]), reinterpret_cast<double*>(c->X[1]), reinterpret_cast<double*>(c->X[2])};
    for (int s = 0; s < nsteps; ++s) {
        // tracers feel the B of the state at the start of the step (t_n): either a separate inverse transform now, or
        // (AB2 + fused sweep) the real-space B that sweep S3 of this step's right-hand side produces anyway
        if (tracers && !emit) {
            if (int rc = tracers_real_B(c, Breal)) return rc;
            tracers_push_with(c, Breal, 1);
        }
        if (c->integrator == 0) {                       // Adams-Bashforth 2, Euler start (R6)
            rhs_spectral(c, c->U, nullptr, c->have_old ? 2 : 1, emit ? Breal : nullptr);
            if (emit) tracers_push_with(c, Breal, 1);
            c->have_old = true;
        } else {
            // RK4 and the predictor-corrector (Heun: U* = U + dt R(U); U+ = U + dt/2 (R(U) + R(U*))) in low-storage
            // form: each stage's assembly pass also accumulates the slope and forms the next stage state (StageUpdate);
            // U0 lives in the R^old buffers, the accumulator in Y
            const double dt = c->dt;
            const double rk4[4][2] = {{0.5 * dt, dt / 6.0}, {0.5 * dt, dt / 3.0}, {dt, dt / 3.0}, {0.0, dt / 6.0}};
            const double heun[2][2] = {{dt, 0.5 * dt}, {0.0, 0.5 * dt}};
            const int ns = c->integrator == 1 ? 4 : 2;
            for (int k = 0; k < ns; ++k) {
                StageUpdate sg;
                std::memset(&sg, 0, sizeof(sg));
                for (int f = 0; f < 8; ++f) { sg.U0[f] = c->Rold[f]; sg.acc[f] = c->Y[f]; }
                sg.c_next = c->integrator == 1 ? rk4[k][0] : heun[k][0];
                sg.b_acc = c->integrator == 1 ? rk4[k][1] : heun[k][1];
                sg.first = k == 0; sg.last = k == ns - 1;
                rhs_spectral(c, c->U, nullptr, 3, nullptr, &sg);
            }
        }
        ++c->step;
    }
    return check_cuda(c, "step");
}

int mhd_get_fields(mhd_ctx* c, int kind, int where, double* const out[8]) {
    if (!c || !out) return MHD_ERR_INVALID_ARG;
    if (!c->bound) return c->fail(MHD_ERR_NOT_BOUND, "mhd_bind has not been called");
    if (!c->have_fields) return c->fail(MHD_ERR_NO_FIELDS, "mhd_set_fields has not been called");
    if ((kind != 0 && kind != 1) || (where != 0 && where != 1)) return c->fail(MHD_ERR_INVALID_ARG, "kind/where");
    if (c->ooc.on) return ooc_get_fields(c, kind, where, out);
    double* real[8];
    for (int i = 0; i < 8; ++i) real[i] = (where == MHD_DEVICE) ? out[i] : reinterpret_cast<double*>(c->W[i]);
    inverse3d(c, 8, c->U, c->W, real, true);
    if (kind == MHD_PRIMITIVE) { mhd_ctx::Scope s(c, F_POINT); launch_cons_to_prim(c->n3(), real, c->gamma, c->st); }
    int rc = copy_out(c, where, real, out);
    return rc ? rc : check_cuda(c, "get_fields");
}

int mhd_diagnostics(mhd_ctx* c, mhd_diag* d, double* spec_kin, double* spec_mag, int nspec) {
    if (!c || !d) return MHD_ERR_INVALID_ARG;
    if (!c->bound) return c->fail(MHD_ERR_NOT_BOUND, "mhd_bind has not been called");
    if (!c->have_fields) return c->fail(MHD_ERR_NO_FIELDS, "mhd_set_fields has not been called");
    const int ns = nspec_of(c->N);
    if (c->ooc.on) return ooc_diagnostics(c, d, spec_kin, spec_mag, nspec);
    if ((spec_kin || spec_mag) && nspec != ns) return c->fail(MHD_ERR_INVALID_ARG, "nspec must equal mhd_nspec(N)");
    const long long n3 = c->n3();
    double* real[8];
    for (int i = 0; i < 8; ++i) real[i] = reinterpret_cast<double*>(c->W[i]);
    inverse3d(c, 8, c->U, c->W, real, true);
    const double* rc8[8];
    for (int i = 0; i < 8; ++i) rc8[i] = real[i];
    { mhd_ctx::Scope s(c, F_DIAG, 2); launch_diag_reduce(n3, rc8, c->gamma, c->scratch, c->res, c->st); }
    {   // max |div~ B|
        SpecGeom g = c->geom(); g.pruned = 1;
        const cd* B[3] = {c->U[5], c->U[6], c->U[7]};
        { mhd_ctx::Scope s(c, F_POINT); launch_divergence(g, B, c->W[8], c->phys(), c->st); }
        const cd* sp[1] = {c->W[8]}; cd* wk[1] = {c->W[8]}; double* ro[1] = {reinterpret_cast<double*>(c->W[8])};
        inverse3d(c, 1, sp, wk, ro, true);
        mhd_ctx::Scope s(c, F_DIAG, 2);
        launch_absmax(n3, ro[0], c->scratch, c->res + 16, c->st);
    }
    if (spec_kin) {
        double* w[3] = {reinterpret_cast<double*>(c->W[9]), reinterpret_cast<double*>(c->W[10]), reinterpret_cast<double*>(c->W[11])};
        { mhd_ctx::Scope s(c, F_POINT); launch_sqrt_rho_u(n3, rc8, w, c->st); }
        const double* wc[3] = {w[0], w[1], w[2]};
        cd* sp[3] = {c->W[9], c->W[10], c->W[11]};
        forward3d(c, 3, wc, sp, c->nyq, false);
        const cd* spc[3] = {sp[0], sp[1], sp[2]}; const cd* nq[3] = {c->nyq[0], c->nyq[1], c->nyq[2]};
        mhd_ctx::Scope s(c, F_DIAG, 2);
        launch_shell_spectrum(c->N, spc, nq, c->scratch, c->res + 64, ns, c->st);
    }
    if (spec_mag) {
        const cd* spc[3] = {c->U[5], c->U[6], c->U[7]};
        mhd_ctx::Scope s(c, F_DIAG, 2);
        launch_shell_spectrum(c->N, spc, nullptr, c->scratch, c->res + 64 + ns, ns, c->st);
    }
    std::vector<double> host(64 + 2 * ns);
    cudaMemcpyAsync(host.data(), c->res, host.size() * sizeof(double), cudaMemcpyDeviceToHost, c->st);
    cudaStreamSynchronize(c->st);
    int rc = check_cuda(c, "diagnostics");
    if (rc) return rc;
    d->t = (double)c->step * c->dt; d->step = c->step;
    d->ke = host[0]; d->me = host[1]; d->ie = host[2]; d->mass = host[3];
    d->mom[0] = host[4]; d->mom[1] = host[5]; d->mom[2] = host[6]; d->etot = host[7];
    d->rho_min = host[8]; d->p_min = host[9]; d->max_divb = host[16];
    if (spec_kin) std::memcpy(spec_kin, host.data() + 64, ns * sizeof(double));
    if (spec_mag) std::memcpy(spec_mag, host.data() + 64 + ns, ns * sizeof(double));
    return MHD_OK;
}

int mhd_fft3d_r2c(mhd_ctx* c, int nfields, const double* const real[], double* const spec[], double* const nyq[], int prune) {
    if (!c || !real || !spec || nfields < 1) return MHD_ERR_INVALID_ARG;
    if (!c->bound) return c->fail(MHD_ERR_NOT_BOUND, "mhd_bind has not been called");
    if (c->ooc.on) return c->fail(MHD_ERR_INVALID_ARG, "mhd_fft3d_* needs an in-core context");
    std::vector<cd*> sp(nfields), nq(nfields);
    for (int f = 0; f < nfields; ++f) { sp[f] = reinterpret_cast<cd*>(spec[f]); nq[f] = nyq ? reinterpret_cast<cd*>(nyq[f]) : nullptr; }
    forward3d(c, nfields, real, sp.data(), (nyq && !prune) ? nq.data() : nullptr, prune != 0);
    return check_cuda(c, "fft3d_r2c");
}
int mhd_fft3d_c2r(mhd_ctx* c, int nfields, double* const spec[], double* const real[], int prune) {
    if (!c || !real || !spec || nfields < 1) return MHD_ERR_INVALID_ARG;
    if (!c->bound) return c->fail(MHD_ERR_NOT_BOUND, "mhd_bind has not been called");
    if (c->ooc.on) return c->fail(MHD_ERR_INVALID_ARG, "mhd_fft3d_* needs an in-core context");
    std::vector<cd*> sp(nfields); std::vector<const cd*> spc(nfields);
    for (int f = 0; f < nfields; ++f) { sp[f] = reinterpret_cast<cd*>(spec[f]); spc[f] = sp[f]; }
    inverse3d(c, nfields, spc.data(), sp.data(), real, prune != 0);
    return check_cuda(c, "fft3d_c2r");
}

// 12 particle arrays (two sets: the spatial sort ping-pongs), 2 id arrays, key + rank, 2^20 histogram bins
static size_t tracer_hist_bytes() { return align_up(((size_t)1 << 20) * sizeof(unsigned)); }
size_t mhd_tracers_field_bytes(const mhd_ctx* c) {
    if (!c || !c->ooc.on) return 0;
    return 4 * align_up((size_t)c->n3() * sizeof(double));
}
size_t mhd_tracers_bytes(long long np) {
    if (np <= 0) return 0;
    return 14 * align_up((size_t)np * sizeof(double)) + 2 * align_up((size_t)np * sizeof(unsigned)) + tracer_hist_bytes();
}

int mhd_tracers_bind(mhd_ctx* c, long long np, void* dev_buffer, size_t bytes) {
    if (!c || np < 0) return MHD_ERR_INVALID_ARG;
    if (!c->bound) return c->fail(MHD_ERR_NOT_BOUND, "mhd_bind has not been called");
    if (c->ooc.on && c->ooc.world > 1) return c->fail(MHD_ERR_INVALID_ARG, "tracers are not available on a decomposed context");
    c->tr = mhd_ctx::Tracers();
    if (np == 0) return MHD_OK;
    if (!dev_buffer || ((uintptr_t)dev_buffer & 255) != 0) return c->fail(MHD_ERR_INVALID_ARG, "tracer buffer must be 256-byte aligned");
    if (bytes < mhd_tracers_bytes(np) + mhd_tracers_field_bytes(c)) return c->fail(MHD_ERR_NOMEM, "tracer buffer too small");
    if (np >= ((long long)1 << 32)) return c->fail(MHD_ERR_INVALID_ARG, "at most 2^32 - 1 tracers");
    const size_t stride = align_up((size_t)np * sizeof(double)), istride = align_up((size_t)np * sizeof(unsigned));
    char* b = static_cast<char*>(dev_buffer);
    for (int d = 0; d < 3; ++d) {
        c->tr.pos[d] = reinterpret_cast<double*>(b + (size_t)d * stride);
        c->tr.vel[d] = reinterpret_cast<double*>(b + (size_t)(3 + d) * stride);
    }
    for (int f = 0; f < 6; ++f) c->tr.alt[f] = reinterpret_cast<double*>(b + (size_t)(6 + f) * stride);
    c->tr.id = reinterpret_cast<long long*>(b + 12 * stride);
    c->tr.alt_id = reinterpret_cast<long long*>(b + 13 * stride);
    c->tr.key = reinterpret_cast<unsigned*>(b + 14 * stride);
    c->tr.rank = reinterpret_cast<unsigned*>(b + 14 * stride + istride);
    c->tr.hist = reinterpret_cast<unsigned*>(b + 14 * stride + 2 * istride);
    if (c->ooc.on)          // chunked context: the real-space field copies follow the particle storage
        for (int f = 0; f < 4; ++f)
            c->tr.field[f] = reinterpret_cast<double*>(b + mhd_tracers_bytes(np) + (size_t)f * align_up((size_t)c->n3() * sizeof(double)));
    c->tr.np = np;
    return MHD_OK;
}

int mhd_tracers_set(mhd_ctx* c, int where, const double* const pos[3], const double* const vel[3]) {
    if (!c || !pos) return MHD_ERR_INVALID_ARG;
    if (!c->bound) return c->fail(MHD_ERR_NOT_BOUND, "mhd_bind has not been called");
    if (c->tr.np <= 0) return c->fail(MHD_ERR_NOT_BOUND, "mhd_tracers_bind has not been called");
    if (where != 0 && where != 1) return c->fail(MHD_ERR_INVALID_ARG, "where");
    if (!vel && !c->have_fields) return c->fail(MHD_ERR_NO_FIELDS, "initial tracer velocity needs mhd_set_fields first");
    const size_t bytes = (size_t)c->tr.np * sizeof(double);
    const cudaMemcpyKind kind = where == MHD_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
    for (int d = 0; d < 3; ++d) {
        if (!pos[d] || (vel && !vel[d])) return c->fail(MHD_ERR_INVALID_ARG, "null tracer array");
        cudaMemcpyAsync(c->tr.pos[d], pos[d], bytes, kind, c->st);
        if (vel) cudaMemcpyAsync(c->tr.vel[d], vel[d], bytes, kind, c->st);
    }
    { mhd_ctx::Scope s(c, F_TRACERS, 2); launch_tracer_wrap(tracer_args(c, nullptr, 0), c->st); launch_tracer_iota(c->tr.np, c->tr.id, c->st); }
    c->tr.sorted = false; c->tr.since_sort = 0;
    if (!vel && c->ooc.on) {     // chunked context: real-space rho, m through the slab stage into the tracers' field arrays
        double* out[8] = {c->tr.field[0], c->tr.field[1], c->tr.field[2], c->tr.field[3], nullptr, nullptr, nullptr, nullptr};
        if (int rc = ooc_real_fields(c, out)) return rc;
        const double* m[3] = {c->tr.field[1], c->tr.field[2], c->tr.field[3]};
        mhd_ctx::Scope s(c, F_TRACERS);
        launch_tracer_init_velocity(tracer_args(c, nullptr, 0), c->tr.field[0], m, c->st);
    } else if (!vel) {      // v0 = CIC of u = m/rho (L241): real-space rho, m of the current state -> X[0..3]
        const cd* spec[4] = {c->U[0], c->U[1], c->U[2], c->U[3]};
        cd* work[4] = {c->X[0], c->X[1], c->X[2], c->X[3]};
        double* real[4];
        for (int f = 0; f < 4; ++f) real[f] = reinterpret_cast<double*>(c->X[f]);
        inverse3d(c, 4, spec, work, real, true);
        const double* m[3] = {real[1], real[2], real[3]};
        mhd_ctx::Scope s(c, F_TRACERS);
        launch_tracer_init_velocity(tracer_args(c, nullptr, 0), real[0], m, c->st);
    }
    if (c->opt_tracer_sort > 0) tracers_sort(c);
    if (where == MHD_HOST) cudaStreamSynchronize(c->st);
    int rc = check_cuda(c, "tracers_set");
    if (rc) return rc;
    c->tr.set = true;
    return MHD_OK;
}

int mhd_tracers_get(mhd_ctx* c, int where, double* const pos[3], double* const vel[3]) {
    if (!c) return MHD_ERR_INVALID_ARG;
    if (!c->bound) return c->fail(MHD_ERR_NOT_BOUND, "mhd_bind has not been called");
    if (!tracers_active(c)) return c->fail(MHD_ERR_NO_FIELDS, "mhd_tracers_set has not been called");
    if (where != 0 && where != 1) return c->fail(MHD_ERR_INVALID_ARG, "where");
    const size_t bytes = (size_t)c->tr.np * sizeof(double);
    const cudaMemcpyKind kind = where == MHD_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
    for (int d = 0; d < 3; ++d) {
        const double* src[2] = {c->tr.pos[d], c->tr.vel[d]};
        double* dst[2] = {pos ? pos[d] : nullptr, vel ? vel[d] : nullptr};
        for (int k = 0; k < 2; ++k) {
            if (!dst[k]) continue;
            if (!c->tr.sorted) { cudaMemcpyAsync(dst[k], src[k], bytes, kind, c->st); continue; }
            // storage is in sorted order: out[id[m]] = in[m], straight into device output or through the spare set
            double* tmp = where == MHD_DEVICE ? dst[k] : c->tr.alt[0];
            { mhd_ctx::Scope s(c, F_TRACERS); launch_tracer_unpermute(c->tr.np, c->tr.id, src[k], tmp, c->st); }
            if (where == MHD_HOST) cudaMemcpyAsync(dst[k], tmp, bytes, cudaMemcpyDeviceToHost, c->st);
        }
    }
    if (where == MHD_HOST) cudaStreamSynchronize(c->st);
    return check_cuda(c, "tracers_get");
}

int mhd_tracers_push(mhd_ctx* c, int nsteps) {
    if (!c || nsteps < 0) return MHD_ERR_INVALID_ARG;
    if (!c->bound) return c->fail(MHD_ERR_NOT_BOUND, "mhd_bind has not been called");
    if (!c->have_fields) return c->fail(MHD_ERR_NO_FIELDS, "mhd_set_fields has not been called");
    if (!tracers_active(c)) return c->fail(MHD_ERR_NO_FIELDS, "mhd_tracers_set has not been called");
    double* Breal[3];
    if (int rc = tracers_real_B(c, Breal)) return rc;
    tracers_push_with(c, Breal, nsteps);
    return check_cuda(c, "tracers_push");
}

int mhd_dist_config(mhd_ctx* c, int rank, int world) {
    if (!c) return MHD_ERR_INVALID_ARG;
    if (!c->bound) return c->fail(MHD_ERR_NOT_BOUND, "mhd_bind has not been called");
    return ooc_dist_config(c, rank, world);
}
int mhd_dist_phase(mhd_ctx* c, int phase, int arg) {
    if (!c) return MHD_ERR_INVALID_ARG;
    if (!c->bound) return c->fail(MHD_ERR_NOT_BOUND, "mhd_bind has not been called");
    if (!c->ooc.on) return c->fail(MHD_ERR_INVALID_ARG, "not a chunked-pipeline context");
    if (phase != MHD_DIST_PHASE_STORE && !c->have_fields) return c->fail(MHD_ERR_NO_FIELDS, "mhd_set_fields has not been called");
    return ooc_dist_phase(c, phase, arg);
}
int mhd_dist_counts(mhd_ctx* c, int dir, int nf, long long* send, long long* recv) {
    if (!c || !c->bound || !c->ooc.on) return MHD_ERR_INVALID_ARG;
    return ooc_dist_counts(c, dir, nf, send, recv);
}
int mhd_dist_pack(mhd_ctx* c, int dir, int nf, double* buf) {
    if (!c || !c->bound || !c->ooc.on) return MHD_ERR_INVALID_ARG;
    return ooc_dist_pack(c, dir, nf, buf, 0);
}
int mhd_dist_unpack(mhd_ctx* c, int dir, int nf, const double* buf) {
    if (!c || !c->bound || !c->ooc.on) return MHD_ERR_INVALID_ARG;
    return ooc_dist_pack(c, dir, nf, const_cast<double*>(buf), 1);
}
int mhd_dist_peers(mhd_ctx* c, const long long* delta_bytes) {
    if (!c || !c->bound || !c->ooc.on) return MHD_ERR_INVALID_ARG;
    return ooc_dist_peers(c, delta_bytes);
}
int mhd_dist_enable_peer_access(mhd_ctx* c, int peer_device) {
    if (!c) return MHD_ERR_INVALID_ARG;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return c->fail(MHD_ERR_CUDA, "no current CUDA device"); }
    if (peer_device == dev) return MHD_OK;
    int can = 0;
    if (cudaDeviceCanAccessPeer(&can, dev, peer_device) != cudaSuccess || !can) {
        cudaGetLastError();
        return c->fail(MHD_ERR_CUDA, "no peer access between the two devices");
    }
    const cudaError_t e = cudaDeviceEnablePeerAccess(peer_device, 0);
    if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) return c->fail(MHD_ERR_CUDA, cudaGetErrorString(e));
    cudaGetLastError();
    return MHD_OK;
}
int mhd_dist_ranges(mhd_ctx* c, int rank, int* ky_lo, int* ky_hi, int* z_lo, int* z_hi) {
    if (!c || !c->bound || !c->ooc.on || rank < 0 || rank >= c->ooc.world) return MHD_ERR_INVALID_ARG;
    if (ky_lo) *ky_lo = c->ooc.ky_lo(rank);
    if (ky_hi) *ky_hi = c->ooc.ky_lo(rank + 1);
    if (z_lo) *z_lo = c->ooc.z_lo(rank, c->N);
    if (z_hi) *z_hi = c->ooc.z_lo(rank + 1, c->N);
    return MHD_OK;
}

long long mhd_launch_count(const mhd_ctx* c) { return c ? c->launches : 0; }

int mhd_transfer_bytes(const mhd_ctx* c, long long* h2d, long long* d2h) {
    if (!c) return MHD_ERR_INVALID_ARG;
    if (h2d) *h2d = c->ooc.h2d_bytes;
    if (d2h) *d2h = c->ooc.d2h_bytes;
    return MHD_OK;
}

int mhd_profile_enable(mhd_ctx* c, int on) {
    if (!c) return MHD_ERR_INVALID_ARG;
    if (c->bound) c->drain_profile();
    c->prof = on != 0;
    for (int i = 0; i < F_COUNT; ++i) { c->fam_ms[i] = 0; c->fam_n[i] = 0; }
    return MHD_OK;
}
int mhd_profile_get(mhd_ctx* c, int max_entries, const char** names, double* ms, long long* launches) {
    if (!c) return MHD_ERR_INVALID_ARG;
    c->drain_profile();
    int n = 0;
    for (int i = 0; i < F_COUNT && n < max_entries; ++i, ++n) {
        if (names) names[n] = family_name(i);
        if (ms) ms[n] = c->fam_ms[i];
        if (launches) launches[n] = c->fam_n[i];
    }
    return n;
}

const char* mhd_last_error(const mhd_ctx* c) { return c ? c->err.c_str() : "null context"; }

int mhd_destroy(mhd_ctx* c) {
    if (!c) return MHD_OK;
    if (c->bound) c->drain_profile();
    ooc_destroy(c);
    for (auto e : c->pool) cudaEventDestroy(e);
    delete c;
    return MHD_OK;
}

}  // extern "C"

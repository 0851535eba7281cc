// ctx.h — the solver context behind the opaque mhd_ctx of include/mhd.h (internal to libmhd).
#pragma once
#include "../../include/mhd.h"
#include "../../include/mhd_bench.h"
#include "kernels.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

using namespace mhd;

enum Family { F_STRIDED_INV = 0, F_STRIDED_FWD, F_X_FUSED, F_X_C2R, F_X_R2C, F_FLUX, F_CURRENT, F_ASSEMBLE, F_AXPBY,
              F_POINT, F_DIAG, F_TRACERS, F_S5, F_COUNT };
inline const char* family_name(int f) {
    static const char* names[F_COUNT] = {"strided_inverse", "strided_forward", "x_fused", "x_c2r", "x_r2c", "flux_real",
                                         "build_current", "assemble", "axpby", "pointwise_misc", "diagnostics", "tracers",
                                         "forward_z_assemble"};
    return names[f];
}

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

constexpr int NFIELD_BUFS = 48;   // U 8, Rold 8, W 16, X 8, Y 8

struct Layout {
    size_t field_bytes, tw_off, ftw_off, field_off, nyq_off, nyq_bytes, scratch_off, scratch_bytes, res_off, total;
};
inline int nspec_of(int N) { return (int)std::ceil(std::sqrt(3.0) * N / 2.0) + 1; }
inline Layout make_layout(int N) {
    Layout l;
    l.field_bytes = (size_t)N * N * N * sizeof(double);
    size_t off = 0;
    l.tw_off = off; off += align_up((size_t)N * sizeof(cd));
    l.ftw_off = off; off += align_up((size_t)(4 * N + 64) * sizeof(cd));
    l.field_off = off; off += (size_t)NFIELD_BUFS * align_up(l.field_bytes);
    l.nyq_bytes = align_up((size_t)N * N * 8 * sizeof(cd));
    l.nyq_off = off; off += 3 * l.nyq_bytes;
    l.scratch_bytes = align_up((size_t)diag_scratch_doubles(nspec_of(N)) * sizeof(double));
    l.scratch_off = off; off += l.scratch_bytes;
    l.res_off = off; off += align_up((size_t)(64 + 2 * nspec_of(N)) * sizeof(double));
    l.total = off;
    return l;
}
inline bool valid_N(int N) { return N >= 16 && N <= 1024 && (N & (N - 1)) == 0; }

struct mhd_ctx {
    int N = 0;
    double L = 0, gamma = 0, mu = 0, eta = 0, dt = 0;
    double cs2 = 0, f0 = 0;          // variants: barotropic sound speed squared, ABC forcing amplitude
    int kf = 1, evolve = 3;          // forcing mode number, evolved equation subsets
    bool bound = false, have_fields = false, have_old = false;
    cudaStream_t st = nullptr;
    unsigned flags = 0;
    int opt_fused = 1, opt_prune = 1, opt_fuse_current = 1, integrator = 0, opt_stress = 0, opt_fuse_assemble = 0;
    long long step = 0;
    long long launches = 0;
    std::string err;
    // device storage (inside the caller's workspace)
    cd* tw = nullptr;
    cd* ftw = nullptr;     // lane-contiguous tables of the fused x sweep
    alignas(64) unsigned char tmaps[4 * 128];   // CUtensorMap x 4 over the field buffers (TMA-fed strided passes)
    StridedTma tma;
    int opt_tma = 0;       // MHD_OPT_TMA
    long long tma_launches = 0, s5_launches = 0;      // mhd_alt_launch_count
    int s5_ok[3] = {-1, -1, -1};                      // one-launch S5, variant v: clusters can be co-scheduled (-1 = not asked yet)
    cd *U[8], *Rold[8], *W[16], *X[8], *Y[8], *nyq[3];
    double *scratch = nullptr, *res = nullptr;
    // chunked ("out-of-core") pipeline, see ooc.cu
    struct Ooc {
        static constexpr int NBUF = 3;
        bool on = false, state_host = false, work_host = false;
        int nzc = 0, nyc = 0, nxp = 0;           // compact extents: 2kc+1, 2kc+1, kc+1 rounded up to 8
        cd *Uc[8], *Rc[8];                       // compact state / history [nzc][nyc][nxp]
        cd* Ac[8] = {};                          // MHD_FLAG_STAGE_STORAGE: accumulator of the multi-stage integrators
        bool stage_storage = false;
        // work arrays between the z and y passes.  Unified layout (one context holds everything): WzB = WzS = [N][nyc][nxp].
        // Per-rank layout (MHD_FLAG_RANKS, `split`): WzB = [N][ny_max][nxp] holds all z of the rank's ky share (stages A, C),
        // WzS = [nz_max][nyc][nxp] all ky of its z share (stage B); the state arrays are [nzc][ny_max][nxp]
        cd *WzB[16], *WzS[16];
        bool split = false;
        int ny_max = 0, nz_max = 0;
        int yoff() const { return split ? ky_lo(rank) : 0; }                       // first ky / z index that is stored
        int zoff(int N) const { return split ? z_lo(rank, N) : 0; }
        long long bstride() const { return (long long)(split ? ny_max : nyc) * nxp; }   // z stride of brick-shaped arrays
        char* stage = nullptr;                   // NBUF staging sets (one big set when nothing lives on the host)
        size_t stage_bytes = 0;                  // bytes of one set
        int nbuf = 1;
        int brick_max = 0, slab_max = 0;         // chunk-size caps set by options (0 = as large as the staging allows)
        cudaStream_t s_in = nullptr, s_out = nullptr;
        cudaEvent_t ev_h2d[NBUF], ev_comp[NBUF], ev_d2h[NBUF], ev_start = nullptr;
        double *part_diag = nullptr, *part_max = nullptr, *part_spec = nullptr;
        long long h2d_bytes = 0, d2h_bytes = 0;
        // slab decomposition over `world` GPUs: this rank owns the compact ky
        // range [ky_lo(rank), ky_lo(rank+1)) for the brick stages and the z planes [z_lo(rank), z_lo(rank+1)) for the slab
        // stage; the exchange between them is done by the caller (all-to-all) on packed buffers
        int rank = 0, world = 1;
        // direct exchange: peer_delta[s] = (rank s's workspace base) - (this rank's), in complex elements; the z passes and
        // the forward y pass then store every row straight into its owner's work arrays (no pack / collective / unpack)
        bool direct = false, direct_active = false;
        long long peer_delta[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        int ky_lo(int r) const { return (int)((long long)nyc * r / world); }
        int z_lo(int r, int N) const { return (int)((long long)N * r / world); }
    } ooc;
    // tracer particles (tracers.cu): caller-provided device storage, 6 arrays of np doubles
    struct Tracers {
        long long np = 0;
        bool set = false;
        double *pos[3] = {nullptr, nullptr, nullptr}, *vel[3] = {nullptr, nullptr, nullptr};
        // spatial sort: second set of arrays (ping-pong), particle ids, counting-sort scratch
        double* alt[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
        long long *id = nullptr, *alt_id = nullptr;
        unsigned *hist = nullptr, *key = nullptr, *rank = nullptr;
        double* field[4] = {nullptr, nullptr, nullptr, nullptr};   // chunked contexts: real-space field copies (B; rho, m)
        bool sorted = false;           // storage order != id order
        int since_sort = 0;            // pushes since the last sort
    } tr;
    int opt_tracer_sort = 32;          // re-sort the tracers every this many pushes (0 = never sort)
    // profiling
    bool prof = false;
    struct Rec { int fam; cudaEvent_t a, b; };
    std::vector<Rec> recs;
    std::vector<cudaEvent_t> pool;
    double fam_ms[F_COUNT] = {0};
    long long fam_n[F_COUNT] = {0};

    int fail(int code, const std::string& m) { err = m; return code; }
    int hx() const { return N / 2; }
    int kc() const { return N / 3; }
    long long n3() const { return (long long)N * N * N; }
    Phys phys() const { return Phys{2.0 * M_PI / L, gamma, mu, eta, cs2, f0, kf, evolve}; }
    SpecGeom geom() const { return SpecGeom{N, N / 2, N / 3, opt_prune}; }

    cudaEvent_t get_event() {
        if (!pool.empty()) { cudaEvent_t e = pool.back(); pool.pop_back(); return e; }
        cudaEvent_t e; cudaEventCreate(&e); return e;
    }
    struct Scope {
        mhd_ctx* c; int fam; cudaEvent_t a = nullptr;
        Scope(mhd_ctx* c_, int fam_, int nlaunch = 1) : c(c_), fam(fam_) {
            c->launches += nlaunch; c->fam_n[fam] += nlaunch;
            if (c->prof) { a = c->get_event(); cudaEventRecord(a, c->st); }
        }
        ~Scope() {
            if (a) { cudaEvent_t b = c->get_event(); cudaEventRecord(b, c->st); c->recs.push_back({fam, a, b}); }
        }
    };
    void drain_profile() {
        if (recs.empty()) return;
        cudaStreamSynchronize(st);
        for (auto& r : recs) {
            float ms = 0; cudaEventElapsedTime(&ms, r.a, r.b);
            fam_ms[r.fam] += ms; pool.push_back(r.a); pool.push_back(r.b);
        }
        recs.clear();
    }
};

inline int check_cuda(mhd_ctx* c, const char* what) {
    cudaError_t e = cudaGetLastError();
    const std::string cfg = kernel_config_error();      // a failed shared-memory / cluster opt-in of this thread, if any
    if (e != cudaSuccess) return c->fail(MHD_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e) + (cfg.empty() ? "" : " [" + cfg + "]"));
    if (!cfg.empty()) return c->fail(MHD_ERR_CUDA, std::string(what) + ": " + cfg);
    return MHD_OK;
}


// ---- shared between mhd_api.cu and ooc.cu -----------------------------------------------------------------------
// sweep S3 on `nlines` consecutive lines (in place allowed): C2R of 11 fields, flux products, R2C of 16 products
void run_x_fused(mhd_ctx* c, cd* const in[11], cd* const out[16], long long nlines, double* const breal[3] = nullptr);

size_t ooc_workspace_bytes(int N, unsigned flags);
size_t ooc_pinned_bytes(int N, unsigned flags);
int ooc_bind(mhd_ctx* c, char* base, size_t bytes, char* pinned, size_t pinned_bytes);
void ooc_destroy(mhd_ctx* c);
int ooc_set_fields(mhd_ctx* c, int kind, int where, const double* const f[8]);
int ooc_get_fields(mhd_ctx* c, int kind, int where, double* const out[8]);
int ooc_rhs(mhd_ctx* c, int where, double* const out[8]);
int ooc_step(mhd_ctx* c, int nsteps);
int ooc_real_fields(mhd_ctx* c, double* const out[8]);
int ooc_diagnostics(mhd_ctx* c, mhd_diag* d, double* spec_kin, double* spec_mag, int nspec);
int ooc_dist_config(mhd_ctx* c, int rank, int world);
int ooc_dist_phase(mhd_ctx* c, int phase, int arg);
int ooc_dist_counts(mhd_ctx* c, int dir, int nf, long long* send, long long* recv);
int ooc_dist_pack(mhd_ctx* c, int dir, int nf, double* buf, int unpack);
int ooc_dist_peers(mhd_ctx* c, const long long* delta_bytes);

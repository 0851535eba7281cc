// ooc.cu — the chunked ("out-of-core") pipeline: SURVEY.md §8(a) row 9, Sec. VII-C (L333-343, L375-379).
//
// The paper lets CUDA unified memory page a working set larger than device memory in and out on demand and finds the
// step an order of magnitude slower than in core (L379).  Here the placement is explicit and the traffic minimal:
//   * storage is COMPACT: the state U^ and the history R^old hold only the (2kc+1)^2 (kc+1) modes inside the 2/3 mask
//     ([kz_c][ky_c][kx_c], 30 % of a full field), the work fields between the z and the y passes hold all N planes in z
//     but only the retained ky, kx ([z][ky_c][kx_c], 45 %);
//   * each class lives either in device memory or in PINNED HOST memory (MHD_FLAG_STATE_ON_HOST, MHD_FLAG_WORK_ON_HOST);
//   * a 3-D transform needs one whole axis at a time (L335, L375), so the step is three chunked stages:
//       A  bricks (a range of ky x all kz x all kx):  U^ -> J^ on load, inverse z pass            -> work[0..10]
//       B  slabs  (a range of z planes):              inverse y, fused x sweep (C2R, fluxes, R2C), forward y -> work[0..15]
//       C  bricks:                                    forward z, assembly of R^, explicit update   -> U^, R^old
//     every chunk of a host-resident class is copied into one of NBUF device staging sets on a copy-in stream,
//     processed on the solver's stream and copied back on a copy-out stream (events order the three), so that PCIe
//     transfers in both directions overlap the kernels;
//   * the kernels are the same templates as in core (strided_kernel<.., GEN = true>, the fused x sweep, the spectral
//     kernels with compact-brick geometry): only data placement changes, results agree with the in-core path to roundoff.
// With nothing on the host the same pipeline is a compact in-core mode: 1024^3 needs ~105 GB and runs without PCIe.
#include "ctx.h"

#include <utility>

namespace {

typedef mhd_ctx::Ooc Ooc;
constexpr int NBUF = Ooc::NBUF;

struct OocSizes {
    int kc, nzc, nyc, nxp, hx;
    size_t celems, welems, selems;   // elements of one compact state / one brick-shaped work / one slab-shaped work array
    size_t cbytes, wbytes, sbytes;
    int ranks, ny_max, nz_max;       // per-rank storage (MHD_FLAG_RANKS): shares of the ky and z axes
    size_t slab_off;
    size_t tw_off, ftw_off, state_off, work_off, stage_off, stage_total, part_off, part_bytes, res_off, total;
    size_t per_ky, per_z;         // staging bytes per ky column of a brick / per z plane of a slab
    bool state_host, work_host;
    int nstate;                   // compact state-shaped arrays: U^ 8 + R^old 8 (+ 8 accumulators with MHD_FLAG_STAGE_STORAGE)
    size_t pinned_total;
};

bool flags_ok(unsigned flags) {
    if (!(flags & MHD_FLAG_OUT_OF_CORE)) return false;
    return true;
}

// all sizes of the chunked pipeline for grid N and placement flags; budget (MiB) bounds the total device workspace
bool ooc_sizes(int N, unsigned flags, OocSizes& s) {
    if (!valid_N(N) || !flags_ok(flags)) return false;
    s.kc = N / 3; s.nzc = 2 * s.kc + 1; s.nyc = s.nzc; s.nxp = (s.kc + 1 + 7) / 8 * 8; s.hx = N / 2;
    s.state_host = (flags & MHD_FLAG_STATE_ON_HOST) != 0;
    s.work_host = (flags & MHD_FLAG_WORK_ON_HOST) != 0;
    s.nstate = (flags & MHD_FLAG_STAGE_STORAGE) ? 24 : 16;
    s.ranks = (int)((flags >> 4) & 7u) + 1;
    if (s.ranks > 1 && (s.state_host || s.work_host || s.ranks > s.nyc || s.ranks > N)) return false;
    s.ny_max = (s.nyc + s.ranks - 1) / s.ranks; s.nz_max = (N + s.ranks - 1) / s.ranks;
    s.celems = (size_t)s.nzc * s.ny_max * s.nxp; s.welems = (size_t)N * s.ny_max * s.nxp;
    s.selems = s.ranks > 1 ? (size_t)s.nz_max * s.nyc * s.nxp : 0;
    s.cbytes = align_up(s.celems * sizeof(cd)); s.wbytes = align_up(s.welems * sizeof(cd)); s.sbytes = align_up(s.selems * sizeof(cd));
    const int ns = nspec_of(N);
    size_t off = 0;
    s.tw_off = off; off += align_up((size_t)N * sizeof(cd));
    s.ftw_off = off; off += align_up((size_t)(4 * N + 64) * sizeof(cd));
    s.state_off = off; if (!s.state_host) off += (size_t)s.nstate * s.cbytes;
    s.work_off = off; if (!s.work_host) off += 16 * s.wbytes;
    s.slab_off = off; off += 16 * s.sbytes;
    s.part_bytes = align_up((size_t)(diag_partial_doubles() + absmax_partial_doubles() + spectrum_partial_doubles(ns)) * sizeof(double));
    s.part_off = off; off += s.part_bytes;
    s.res_off = off; off += align_up((size_t)(64 + 2 * ns) * sizeof(double));
    // staging: per ky column of a brick: 16 z-full work columns (if on host), U and R^old columns (if on host), plus
    // 9 compact columns of scratch (R^ of mhd_rhs / the divergence of mhd_diagnostics); per z plane of a slab: the
    // 16 full-pitch planes of the x sweep plus the compact in (11) and out (16) planes when the work lives on the host
    const size_t col = (size_t)s.nxp * sizeof(cd);
    s.per_ky = ((s.work_host ? 16 * (size_t)N : 0) + (s.state_host ? (size_t)s.nstate * s.nzc : 0) + 9 * (size_t)s.nzc) * col + 64 * 256;
    s.per_z = 16 * (size_t)N * s.hx * sizeof(cd) + (s.work_host ? 27 * (size_t)s.nyc * col : 0) + 64 * 256;
    const size_t min_set = std::max(s.per_ky, s.per_z);
    const size_t want_set = std::max(s.per_ky * (size_t)std::min(s.kc + 1, 16), s.per_z * (size_t)std::min(N, 8));
    const size_t budget = (size_t)(flags >> 8) << 20;
    size_t set = want_set;
    if (budget) {
        if (budget < off + NBUF * min_set) return false;
        set = std::min(want_set * 4, (budget - off) / NBUF / 256 * 256);
    }
    s.stage_off = off; s.stage_total = NBUF * align_up(set); off += s.stage_total;
    s.total = off;
    s.pinned_total = (s.state_host ? (size_t)s.nstate * s.cbytes : 0) + (s.work_host ? 16 * s.wbytes : 0);
    return true;
}

// ---- chunk bookkeeping: staging sets, streams, events --------------------------------------------------------------
struct Chunk {
    int b = 0; char* base = nullptr; size_t off = 0, cap = 0; bool overflow = false;
    cd* alloc(size_t elems) {
        cd* p = reinterpret_cast<cd*>(base + off);
        off += align_up(elems * sizeof(cd));
        if (off > cap) overflow = true;
        return p;
    }
};

void stage_begin(mhd_ctx* c) {
    Ooc& o = c->ooc;
    cudaEventRecord(o.ev_start, c->st);
    cudaStreamWaitEvent(o.s_in, o.ev_start, 0);
    cudaStreamWaitEvent(o.s_out, o.ev_start, 0);
}
// staging set of chunk i; `h2d`: the chunk starts with copies on the copy-in stream
Chunk chunk_begin(mhd_ctx* c, int i, bool h2d) {
    Ooc& o = c->ooc;
    Chunk ch;
    ch.b = i % o.nbuf; ch.base = o.stage + (size_t)ch.b * o.stage_bytes; ch.cap = o.stage_bytes;
    if (h2d) {      // the set is free once chunk i - nbuf has been computed and copied out
        cudaStreamWaitEvent(o.s_in, o.ev_comp[ch.b], 0);
        cudaStreamWaitEvent(o.s_in, o.ev_d2h[ch.b], 0);
    } else {
        cudaStreamWaitEvent(c->st, o.ev_d2h[ch.b], 0);
    }
    return ch;
}
void chunk_h2d_done(mhd_ctx* c, const Chunk& ch) {
    Ooc& o = c->ooc;
    cudaEventRecord(o.ev_h2d[ch.b], o.s_in);
    cudaStreamWaitEvent(c->st, o.ev_h2d[ch.b], 0);
}
void chunk_comp_done(mhd_ctx* c, const Chunk& ch, bool d2h) {
    Ooc& o = c->ooc;
    cudaEventRecord(o.ev_comp[ch.b], c->st);
    if (d2h) cudaStreamWaitEvent(o.s_out, o.ev_comp[ch.b], 0);
}
void chunk_d2h_done(mhd_ctx* c, const Chunk& ch) { cudaEventRecord(c->ooc.ev_d2h[ch.b], c->ooc.s_out); }
// the solver's stream has seen everything the stage wrote to host arrays
void stage_end(mhd_ctx* c) {
    Ooc& o = c->ooc;
    for (int b = 0; b < o.nbuf; ++b) cudaStreamWaitEvent(c->st, o.ev_d2h[b], 0);
}

// 2-D copies in units of complex elements (pitches and width), host <-> device
void h2d_2d(mhd_ctx* c, cd* dst, size_t dpitch, const cd* src, size_t spitch, size_t width, size_t height) {
    cudaMemcpy2DAsync(dst, dpitch * sizeof(cd), src, spitch * sizeof(cd), width * sizeof(cd), height, cudaMemcpyHostToDevice, c->ooc.s_in);
    c->ooc.h2d_bytes += (long long)(width * height * sizeof(cd));
}
void d2h_2d(mhd_ctx* c, cd* dst, size_t dpitch, const cd* src, size_t spitch, size_t width, size_t height) {
    cudaMemcpy2DAsync(dst, dpitch * sizeof(cd), src, spitch * sizeof(cd), width * sizeof(cd), height, cudaMemcpyDeviceToHost, c->ooc.s_out);
    c->ooc.d2h_bytes += (long long)(width * height * sizeof(cd));
}
void h2d_1d(mhd_ctx* c, void* dst, const void* src, size_t bytes) {
    cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, c->ooc.s_in);
    c->ooc.h2d_bytes += (long long)bytes;
}
void d2h_1d(mhd_ctx* c, void* dst, const void* src, size_t bytes) {
    cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, c->ooc.s_out);
    c->ooc.d2h_bytes += (long long)bytes;
}

// ky ranges of the bricks: never across the split between ky >= 0 (compact 0..kc) and ky < 0 (compact kc+1..2kc)
std::vector<std::pair<int, int>> brick_chunks(const mhd_ctx* c) {
    const Ooc& o = c->ooc;
    OocSizes s; ooc_sizes(c->N, c->flags, s);
    long long nmax = (long long)(o.stage_bytes / s.per_ky);
    const int kc = c->kc();
    if (!o.state_host && !o.work_host) nmax = kc + 1;
    if (o.brick_max > 0) nmax = std::min<long long>(nmax, o.brick_max);
    nmax = std::max<long long>(1, std::min<long long>(nmax, kc + 1));
    std::vector<std::pair<int, int>> v;
    const int ya = o.ky_lo(o.rank), yb = o.ky_lo(o.rank + 1);     // this rank's share (everything when world = 1)
    auto add = [&](int lo, int hi) {
        lo = std::max(lo, ya); hi = std::min(hi, yb);
        for (int y = lo; y < hi; y += (int)nmax) v.push_back({y, (int)std::min<long long>(nmax, hi - y)});
    };
    add(0, kc + 1);
    add(kc + 1, 2 * kc + 1);
    return v;
}
std::vector<std::pair<int, int>> slab_chunks(const mhd_ctx* c) {
    const Ooc& o = c->ooc;
    OocSizes s; ooc_sizes(c->N, c->flags, s);
    long long nmax = (long long)(o.stage_bytes / s.per_z);
    if (o.slab_max > 0) nmax = std::min<long long>(nmax, o.slab_max);
    nmax = std::max<long long>(1, std::min<long long>(nmax, c->N));
    std::vector<std::pair<int, int>> v;
    const int za = o.z_lo(o.rank, c->N), zb = o.z_lo(o.rank + 1, c->N);
    for (int z = za; z < zb; z += (int)nmax) v.push_back({z, (int)std::min<long long>(nmax, zb - z)});
    return v;
}

// general strided pass (kernels_strided.cu, GEN = true): nf fields, rows = the transformed axis, `n_outer` outer indices
// peer_rows (direct exchange of a decomposed context, only while o.direct_active): 1 = the output rows are z planes,
// 2 = compact ky rows; each row is then stored into its owner's workspace
void gen_pass(mhd_ctx* c, int dir, int nf, const cd* const in[], cd* const out[], long long irs, long long ios, int in_rows,
              long long ors, long long oos, int out_rows, int n_outer, int jfirst = -1, int bfirst = 0, int outer_base = 0,
              int peer_rows = 0) {
    StridedArgs a;
    std::memset(&a, 0, sizeof(a));
    for (int f = 0; f < nf; ++f) { a.in[f] = in[f]; a.out[f] = out[f]; }
    a.tw = c->tw; a.kc = c->kc(); a.nfields = nf; a.general = 1;
    a.in_row_stride = irs; a.in_outer_stride = ios; a.in_rows = in_rows;
    a.out_row_stride = ors; a.out_outer_stride = oos; a.out_rows = out_rows;
    a.n_outer = n_outer; a.outer_split = n_outer; a.outer_skip = 0;
    a.ncols = c->kc() + 1;
    a.jfirst = jfirst; a.bfirst = bfirst; a.outer_compact = 1; a.outer_base = outer_base; a.k0 = 2.0 * M_PI / c->L;
    const Ooc& o = c->ooc;
    if (peer_rows && o.direct_active && o.world > 1) {
        a.npeer = o.world;
        for (int s = 0; s <= o.world; ++s) a.peer_lo[s] = peer_rows == 1 ? o.z_lo(s, c->N) : o.ky_lo(s);
        // per-rank storage: the owner's array starts at its own first z plane / ky row
        const long long plane = (long long)o.nyc * o.nxp;
        for (int s = 0; s < o.world; ++s)
            a.peer_delta[s] = o.peer_delta[s] - (o.split ? (peer_rows == 1 ? o.z_lo(s, c->N) * plane : (long long)o.ky_lo(s) * o.nxp) : 0);
    }
    mhd_ctx::Scope s(c, dir > 0 ? F_STRIDED_INV : F_STRIDED_FWD);
    launch_strided(c->N, dir, a, c->st);
}

struct View { cd* p[16]; long long rs = 0; };     // per-field base pointers of a brick + its row stride (outer stride = nxp)

// brick view of `nf` compact state arrays for ky range (y0, ny); host-resident: staged (copied in if `load`)
View state_view(mhd_ctx* c, Chunk& ch, cd* const arr[], int nf, int y0, int ny, bool load) {
    const Ooc& o = c->ooc;
    View v;
    if (o.state_host) {
        v.rs = (long long)ny * o.nxp;
        for (int f = 0; f < nf; ++f) {
            v.p[f] = ch.alloc((size_t)o.nzc * ny * o.nxp);
            if (load && !ch.overflow) h2d_2d(c, v.p[f], (size_t)v.rs, arr[f] + (size_t)y0 * o.nxp, (size_t)o.nyc * o.nxp, (size_t)v.rs, o.nzc);
        }
    } else {
        v.rs = o.bstride();
        for (int f = 0; f < nf; ++f) v.p[f] = arr[f] + (size_t)(y0 - o.yoff()) * o.nxp;
    }
    return v;
}
void state_store(mhd_ctx* c, const View& v, cd* const arr[], int nf, int y0) {
    const Ooc& o = c->ooc;
    if (!o.state_host) return;
    for (int f = 0; f < nf; ++f)
        d2h_2d(c, arr[f] + (size_t)y0 * o.nxp, (size_t)o.nyc * o.nxp, v.p[f], (size_t)v.rs, (size_t)v.rs, o.nzc);
}
View work_view(mhd_ctx* c, Chunk& ch, int nf, int y0, int ny, bool load) {
    const Ooc& o = c->ooc;
    View v;
    if (o.work_host) {
        v.rs = (long long)ny * o.nxp;
        for (int f = 0; f < nf; ++f) {
            v.p[f] = ch.alloc((size_t)c->N * ny * o.nxp);
            if (load && !ch.overflow) h2d_2d(c, v.p[f], (size_t)v.rs, o.WzB[f] + (size_t)y0 * o.nxp, (size_t)o.nyc * o.nxp, (size_t)v.rs, c->N);
        }
    } else {
        v.rs = o.bstride();
        for (int f = 0; f < nf; ++f) v.p[f] = o.WzB[f] + (size_t)(y0 - o.yoff()) * o.nxp;
    }
    return v;
}
void work_store(mhd_ctx* c, const View& v, int nf, int y0) {
    const Ooc& o = c->ooc;
    if (!o.work_host) return;
    for (int f = 0; f < nf; ++f)
        d2h_2d(c, o.WzB[f] + (size_t)y0 * o.nxp, (size_t)o.nyc * o.nxp, v.p[f], (size_t)v.rs, (size_t)v.rs, c->N);
}
SpecGeom brick_geom(const mhd_ctx* c, int y0, int ny, long long wrs, long long srs) {
    SpecGeom g = c->geom();
    g.pruned = 1; g.compact = 1; g.y0 = y0; g.ny = ny;
    g.wsy = c->ooc.nxp; g.wsz = wrs; g.ssy = c->ooc.nxp; g.ssz = srs;
    return g;
}

// where the inverse z pass of a brick writes: its own brick view — or, in the direct exchange with per-rank storage, the
// SLAB-shaped arrays of the z planes' owners (addressed from this rank's slab array; gen_pass adds the owner's offset)
View inverse_z_target(const mhd_ctx* c, const View& w, int y0) {
    const Ooc& o = c->ooc;
    if (!(o.direct_active && o.split)) return w;
    View v;
    v.rs = (long long)o.nyc * o.nxp;
    for (int f = 0; f < 16; ++f) v.p[f] = o.WzS[f] + (size_t)y0 * o.nxp;
    return v;
}

int overflow(mhd_ctx* c) { return c->fail(MHD_ERR_NOMEM, "chunked pipeline: staging set too small for one chunk"); }

// ---- stage A: compact state -> (J^ on load) inverse z pass -> work[0..nf) -----------------------------------------
int stage_inverse_z(mhd_ctx* c, cd* const src[8], bool current) {
    Ooc& o = c->ooc;
    const int nf = current ? 11 : 8;
    stage_begin(c);
    const auto chunks = brick_chunks(c);
    for (size_t i = 0; i < chunks.size(); ++i) {
        const int y0 = chunks[i].first, ny = chunks[i].second;
        Chunk ch = chunk_begin(c, (int)i, o.state_host);
        View u = state_view(c, ch, src, 8, y0, ny, true);
        View w = work_view(c, ch, nf, y0, ny, false);
        if (ch.overflow) return overflow(c);
        if (o.state_host) chunk_h2d_done(c, ch);
        const cd* in[11];
        for (int f = 0; f < 11; ++f) in[f] = u.p[f < 8 ? f : 5];
        const View wo = inverse_z_target(c, w, y0);
        gen_pass(c, +1, nf, in, wo.p, u.rs, o.nxp, 2, wo.rs, o.nxp, 0, ny, current ? 8 : -1, 5, y0, 1);
        chunk_comp_done(c, ch, o.work_host);
        if (o.work_host) { work_store(c, w, nf, y0); chunk_d2h_done(c, ch); }
    }
    stage_end(c);
    return check_cuda(c, "chunked inverse z");
}

// ---- stage B and its relatives: slabs of z planes ---------------------------------------------------------------
enum SlabKind { SLAB_FLUX, SLAB_TO_REAL, SLAB_FROM_REAL };
struct SlabIO {
    int nin = 0, nout = 0;                 // spectral work fields read / written
    int kind = MHD_CONSERVATIVE, where = MHD_HOST;
    const double* const* user_in = nullptr;  // SLAB_FROM_REAL: 8 real fields
    double* const* user_out = nullptr;       // SLAB_TO_REAL: first 8 real fields go here (may be null)
    bool diag = false;                     // SLAB_TO_REAL: accumulate the diagnostics partials (field 8 = div B)
};

int stage_slabs(mhd_ctx* c, SlabKind kind, const SlabIO& io) {
    Ooc& o = c->ooc;
    const int N = c->N, hx = c->hx();
    const size_t plane_c = (size_t)o.nyc * o.nxp;             // one compact z plane (complex elements)
    const size_t plane_r = (size_t)N * N;                     // one real z plane (doubles)
    const bool user_h2d = kind == SLAB_FROM_REAL && io.where == MHD_HOST;
    const bool user_d2h = kind == SLAB_TO_REAL && io.user_out && io.where == MHD_HOST;
    const bool in_copy = (io.nin > 0 && o.work_host) || user_h2d;
    const bool out_copy = (io.nout > 0 && o.work_host) || user_d2h;
    stage_begin(c);
    const auto chunks = slab_chunks(c);
    for (size_t i = 0; i < chunks.size(); ++i) {
        const int z0 = chunks[i].first, zc = chunks[i].second;
        Chunk ch = chunk_begin(c, (int)i, in_copy);
        cd* sb[16];
        const int nsb = kind == SLAB_FLUX ? 16 : std::max(io.nin, 8);
        for (int f = 0; f < nsb; ++f) sb[f] = ch.alloc((size_t)zc * N * hx);
        const cd* in[16]; cd* out[16];
        for (int f = 0; f < io.nin; ++f) {
            if (o.work_host) {
                cd* p = ch.alloc((size_t)zc * plane_c);
                if (!ch.overflow) h2d_1d(c, p, o.WzS[f] + (size_t)z0 * plane_c, (size_t)zc * plane_c * sizeof(cd));
                in[f] = p;
            } else in[f] = o.WzS[f] + (size_t)(z0 - o.zoff(N)) * plane_c;
        }
        // direct exchange with per-rank storage: the forward y pass stores each ky row into its owner's BRICK-shaped array
        const bool to_bricks = io.nout > 0 && kind == SLAB_FLUX && o.direct_active && o.split;
        for (int f = 0; f < io.nout; ++f)
            out[f] = o.work_host ? ch.alloc((size_t)zc * plane_c)
                   : to_bricks ? o.WzB[f] + (size_t)z0 * o.bstride()
                               : o.WzS[f] + (size_t)(z0 - o.zoff(N)) * plane_c;
        if (ch.overflow) return overflow(c);
        if (kind == SLAB_FROM_REAL) {
            for (int f = 0; f < 8; ++f) {
                const double* src = io.user_in[f] + (size_t)z0 * plane_r;
                if (io.where == MHD_HOST) h2d_1d(c, sb[f], src, (size_t)zc * plane_r * sizeof(double));
                else cudaMemcpyAsync(sb[f], src, (size_t)zc * plane_r * sizeof(double), cudaMemcpyDeviceToDevice, c->st);
            }
        }
        if (in_copy) chunk_h2d_done(c, ch);

        double* real[16];
        for (int f = 0; f < nsb; ++f) real[f] = reinterpret_cast<double*>(sb[f]);
        const long long nlines = (long long)zc * N;
        if (io.nin > 0)      // inverse y pass: compact ky rows of the slab -> all N rows at full pitch
            gen_pass(c, +1, io.nin, in, sb, o.nxp, (long long)plane_c, 2, hx, (long long)N * hx, 0, zc);
        if (kind == SLAB_FLUX) {
            run_x_fused(c, sb, sb, nlines);
        } else if (kind == SLAB_TO_REAL) {
            XArgs a; std::memset(&a, 0, sizeof(a));
            for (int f = 0; f < io.nin; ++f) { a.spec_in[f] = sb[f]; a.real_out[f] = real[f]; }
            a.tw = c->tw; a.nlines = nlines; a.nfields = io.nin; a.kmax = c->kc(); a.scale = 1.0 / ((double)N * N * N);
            { mhd_ctx::Scope s(c, F_X_C2R); launch_x_c2r(N, a, c->st); }
            if (io.diag) {
                const double* r8[8];
                for (int f = 0; f < 8; ++f) r8[f] = real[f];
                mhd_ctx::Scope s(c, F_DIAG, 2);
                launch_diag_partial(nlines * N, r8, c->gamma, o.part_diag, i > 0, c->st);
                launch_absmax_partial(nlines * N, real[8], o.part_max, i > 0, c->st);
            }
            if (io.kind == MHD_PRIMITIVE) { mhd_ctx::Scope s(c, F_POINT); launch_cons_to_prim(nlines * N, real, c->gamma, c->st); }
            if (io.user_out && io.where == MHD_DEVICE)
                for (int f = 0; f < 8; ++f)
                    if (io.user_out[f])
                        cudaMemcpyAsync(io.user_out[f] + (size_t)z0 * plane_r, real[f], (size_t)zc * plane_r * sizeof(double), cudaMemcpyDeviceToDevice, c->st);
        } else {             // SLAB_FROM_REAL
            if (io.kind == MHD_PRIMITIVE) { mhd_ctx::Scope s(c, F_POINT); launch_prim_to_cons(nlines * N, real, c->gamma, c->st); }
            XArgs a; std::memset(&a, 0, sizeof(a));
            for (int f = 0; f < 8; ++f) { a.real_in[f] = real[f]; a.spec_out[f] = sb[f]; }
            a.tw = c->tw; a.nlines = nlines; a.nfields = 8; a.kmax = c->kc(); a.scale = 1.0;
            mhd_ctx::Scope s(c, F_X_R2C);
            launch_x_r2c(N, a, c->st);
        }
        if (io.nout > 0)     // forward y pass: all N rows -> the compact ky rows of the slab
            gen_pass(c, -1, io.nout, sb, out, hx, (long long)N * hx, 0, o.nxp, to_bricks ? o.bstride() : (long long)plane_c, 2, zc,
                     -1, 0, 0, 2);
        chunk_comp_done(c, ch, out_copy);
        if (out_copy) {
            if (io.nout > 0 && o.work_host)
                for (int f = 0; f < io.nout; ++f) d2h_1d(c, o.WzS[f] + (size_t)z0 * plane_c, out[f], (size_t)zc * plane_c * sizeof(cd));
            if (user_d2h)
                for (int f = 0; f < 8; ++f)
                    if (io.user_out[f]) d2h_1d(c, io.user_out[f] + (size_t)z0 * plane_r, real[f], (size_t)zc * plane_r * sizeof(double));
            chunk_d2h_done(c, ch);
        }
    }
    stage_end(c);
    return check_cuda(c, "chunked slab stage");
}

// ---- stage C: forward z pass of the 16 products, assembly of R^ and the explicit update (mode 1 Euler, 2 AB2);
//      mode 0 (mhd_rhs): R^ replaces the first 8 work fields and is inverse-z-transformed on the spot.
//      next_inverse (modes 1, 2): stage A of the NEXT step runs on the freshly updated brick while it is still on the
//      device (the z pass is local to a brick), which saves one host->device pass over U^ per step ----------------------
int stage_forward_z_assemble(mhd_ctx* c, int mode, bool next_inverse, const StageUpdate* sg = nullptr) {
    Ooc& o = c->ooc;
    stage_begin(c);
    const auto chunks = brick_chunks(c);
    const bool h2d = o.work_host || o.state_host;
    for (size_t i = 0; i < chunks.size(); ++i) {
        const int y0 = chunks[i].first, ny = chunks[i].second;
        Chunk ch = chunk_begin(c, (int)i, h2d);
        View w = work_view(c, ch, 16, y0, ny, true);
        View u = state_view(c, ch, o.Uc, 8, y0, ny, true);
        View r, acc;
        if (mode != 0) r = state_view(c, ch, o.Rc, 8, y0, ny, mode == 2 || (mode == 3 && !sg->first));
        if (mode == 3) acc = state_view(c, ch, o.Ac, 8, y0, ny, !sg->first);      // (the last stage only reads it)
        if (ch.overflow) return overflow(c);
        if (h2d) chunk_h2d_done(c, ch);
        gen_pass(c, -1, 16, w.p, w.p, w.rs, o.nxp, 0, w.rs, o.nxp, 2, ny);          // in place: rows compacted
        const SpecGeom g = brick_geom(c, y0, ny, w.rs, u.rs);
        {
            mhd_ctx::Scope s(c, F_ASSEMBLE);
            StageUpdate st3 = StageUpdate();
            if (mode == 3) {        // multi-stage integrators: U0 in the R^old arrays, accumulator in Ac (brick views)
                st3 = *sg;
                for (int f = 0; f < 8; ++f) { st3.U0[f] = r.p[f]; st3.acc[f] = acc.p[f]; }
            }
            launch_assemble(g, w.p, u.p, mode != 0 ? r.p : nullptr, mode == 0 ? w.p : nullptr, mode, c->dt, c->phys(), c->st, nullptr,
                            nullptr, mode == 3 ? &st3 : nullptr);
        }
        if (mode == 0) gen_pass(c, +1, 8, w.p, w.p, w.rs, o.nxp, 2, w.rs, o.nxp, 0, ny);
        if (mode != 0 && next_inverse) {
            const cd* in[11];
            for (int f = 0; f < 11; ++f) in[f] = u.p[f < 8 ? f : 5];
            const View wo = inverse_z_target(c, w, y0);
            gen_pass(c, +1, 11, in, wo.p, u.rs, o.nxp, 2, wo.rs, o.nxp, 0, ny, 8, 5, y0, 1);
        }
        const bool d2h = mode == 0 ? o.work_host : (o.state_host || (next_inverse && o.work_host));
        chunk_comp_done(c, ch, d2h);
        if (d2h) {
            if (mode == 0) work_store(c, w, 8, y0);
            else {
                state_store(c, u, o.Uc, 8, y0);
                if (mode != 3 || sg->first) state_store(c, r, o.Rc, 8, y0);
                if (mode == 3 && !sg->last) state_store(c, acc, o.Ac, 8, y0);
                if (next_inverse) work_store(c, w, 11, y0);
            }
            chunk_d2h_done(c, ch);
        }
    }
    stage_end(c);
    return check_cuda(c, "chunked forward z + assembly");
}

// forward z pass of work[0..7] and projection into the compact state (mhd_set_fields)
int stage_forward_z_store(mhd_ctx* c) {
    Ooc& o = c->ooc;
    stage_begin(c);
    const auto chunks = brick_chunks(c);
    for (size_t i = 0; i < chunks.size(); ++i) {
        const int y0 = chunks[i].first, ny = chunks[i].second;
        Chunk ch = chunk_begin(c, (int)i, o.work_host);
        View w = work_view(c, ch, 8, y0, ny, true);
        View u = state_view(c, ch, o.Uc, 8, y0, ny, false);
        if (ch.overflow) return overflow(c);
        if (o.work_host) chunk_h2d_done(c, ch);
        gen_pass(c, -1, 8, w.p, w.p, w.rs, o.nxp, 0, w.rs, o.nxp, 2, ny);
        const SpecGeom g = brick_geom(c, y0, ny, w.rs, u.rs);
        {
            const cd* src[8];
            for (int f = 0; f < 8; ++f) src[f] = w.p[f];
            mhd_ctx::Scope s(c, F_AXPBY);
            launch_copy_masked(g, 8, u.p, src, c->st);
        }
        chunk_comp_done(c, ch, o.state_host);
        if (o.state_host) { state_store(c, u, o.Uc, 8, y0); chunk_d2h_done(c, ch); }
    }
    stage_end(c);
    return check_cuda(c, "chunked forward z + store");
}

// diagnostics, brick part: div~ B^ and the magnetic spectrum from the compact state, inverse z of (U^, div^) -> work[0..8]
int stage_diag_bricks(mhd_ctx* c, bool spec_mag) {
    Ooc& o = c->ooc;
    const int ns = nspec_of(c->N);
    stage_begin(c);
    const auto chunks = brick_chunks(c);
    for (size_t i = 0; i < chunks.size(); ++i) {
        const int y0 = chunks[i].first, ny = chunks[i].second;
        Chunk ch = chunk_begin(c, (int)i, o.state_host);
        View u = state_view(c, ch, o.Uc, 8, y0, ny, true);
        View w = work_view(c, ch, 9, y0, ny, false);
        cd* dv = ch.alloc((size_t)o.nzc * ny * o.nxp);
        if (ch.overflow) return overflow(c);
        if (o.state_host) chunk_h2d_done(c, ch);
        const long long drs = (long long)ny * o.nxp;
        const SpecGeom g = brick_geom(c, y0, ny, drs, u.rs);
        const cd* B[3] = {u.p[5], u.p[6], u.p[7]};
        { mhd_ctx::Scope s(c, F_POINT); launch_divergence(g, B, dv, c->phys(), c->st); }
        if (spec_mag) { mhd_ctx::Scope s(c, F_DIAG); launch_shell_spectrum_compact(g, B, o.part_spec, ns, i > 0, c->st); }
        const cd* in[8];
        for (int f = 0; f < 8; ++f) in[f] = u.p[f];
        gen_pass(c, +1, 8, in, w.p, u.rs, o.nxp, 2, w.rs, o.nxp, 0, ny);
        const cd* din[1] = {dv}; cd* dout[1] = {w.p[8]};
        gen_pass(c, +1, 1, din, dout, drs, o.nxp, 2, w.rs, o.nxp, 0, ny);
        chunk_comp_done(c, ch, o.work_host);
        if (o.work_host) { work_store(c, w, 9, y0); chunk_d2h_done(c, ch); }
    }
    stage_end(c);
    return check_cuda(c, "chunked diagnostics");
}

}  // namespace

// =====================================================================================================================
size_t ooc_workspace_bytes(int N, unsigned flags) {
    OocSizes s;
    return ooc_sizes(N, flags, s) ? s.total : 0;
}
size_t ooc_pinned_bytes(int N, unsigned flags) {
    OocSizes s;
    return ooc_sizes(N, flags, s) ? s.pinned_total : 0;
}

int ooc_bind(mhd_ctx* c, char* base, size_t bytes, char* pinned, size_t pinned_bytes) {
    OocSizes s;
    if (!ooc_sizes(c->N, c->flags, s)) return c->fail(MHD_ERR_INVALID_ARG, "flags / device budget not usable for this N");
    if (bytes < s.total) return c->fail(MHD_ERR_NOMEM, "workspace too small");
    if (s.pinned_total && (!pinned || pinned_bytes < s.pinned_total || ((uintptr_t)pinned & 255)))
        return c->fail(MHD_ERR_NOMEM, "pinned host memory missing, too small or not 256-byte aligned (mhd_pinned_bytes)");
    Ooc& o = c->ooc;
    o.on = true; o.state_host = s.state_host; o.work_host = s.work_host;
    o.nzc = s.nzc; o.nyc = s.nyc; o.nxp = s.nxp;
    c->tw = reinterpret_cast<cd*>(base + s.tw_off);
    c->ftw = reinterpret_cast<cd*>(base + s.ftw_off);
    char* hp = pinned;
    o.stage_storage = s.nstate > 16;
    for (int f = 0; f < s.nstate; ++f) {
        cd*& dst = f < 8 ? o.Uc[f] : (f < 16 ? o.Rc[f - 8] : o.Ac[f - 16]);
        if (s.state_host) { dst = reinterpret_cast<cd*>(hp); hp += s.cbytes; }
        else dst = reinterpret_cast<cd*>(base + s.state_off + (size_t)f * s.cbytes);
    }
    for (int f = 0; f < 16; ++f) {
        if (s.work_host) { o.WzB[f] = reinterpret_cast<cd*>(hp); hp += s.wbytes; }
        else o.WzB[f] = reinterpret_cast<cd*>(base + s.work_off + (size_t)f * s.wbytes);
        o.WzS[f] = s.ranks > 1 ? reinterpret_cast<cd*>(base + s.slab_off + (size_t)f * s.sbytes) : o.WzB[f];
    }
    o.split = s.ranks > 1; o.ny_max = s.ny_max; o.nz_max = s.nz_max;
    o.rank = 0; o.world = s.ranks;            // per-rank storage: mhd_dist_config(rank, ranks) must follow
    o.direct = false;
    const bool any_host = s.state_host || s.work_host;
    o.nbuf = any_host ? NBUF : 1;
    o.stage = base + s.stage_off;
    o.stage_bytes = any_host ? s.stage_total / NBUF : s.stage_total;
    double* part = reinterpret_cast<double*>(base + s.part_off);
    o.part_diag = part; o.part_max = part + diag_partial_doubles(); o.part_spec = o.part_max + absmax_partial_doubles();
    c->scratch = part;
    c->res = reinterpret_cast<double*>(base + s.res_off);
    if (!o.s_in) {
        cudaStreamCreateWithFlags(&o.s_in, cudaStreamNonBlocking);
        cudaStreamCreateWithFlags(&o.s_out, cudaStreamNonBlocking);
        for (int b = 0; b < NBUF; ++b) {
            cudaEventCreateWithFlags(&o.ev_h2d[b], cudaEventDisableTiming);
            cudaEventCreateWithFlags(&o.ev_comp[b], cudaEventDisableTiming);
            cudaEventCreateWithFlags(&o.ev_d2h[b], cudaEventDisableTiming);
        }
        cudaEventCreateWithFlags(&o.ev_start, cudaEventDisableTiming);
    }
    // padding columns / never-written regions must not hold NaN patterns that a masked load could pick up: the kernels
    // only ever touch columns <= kc, so no clearing is required; the compact state is fully written by mhd_set_fields
    launch_twiddle_table(c->N, c->tw, c->st);
    launch_x_fused2_tables(c->N, c->ftw, c->st);
    c->launches += 2;
    return check_cuda(c, "bind (chunked pipeline)");
}

void ooc_destroy(mhd_ctx* c) {
    Ooc& o = c->ooc;
    if (!o.s_in) return;
    cudaStreamSynchronize(o.s_in); cudaStreamSynchronize(o.s_out);
    for (int b = 0; b < NBUF; ++b) { cudaEventDestroy(o.ev_h2d[b]); cudaEventDestroy(o.ev_comp[b]); cudaEventDestroy(o.ev_d2h[b]); }
    cudaEventDestroy(o.ev_start);
    cudaStreamDestroy(o.s_in); cudaStreamDestroy(o.s_out);
    o.s_in = o.s_out = nullptr;
}

int ooc_set_fields(mhd_ctx* c, int kind, int where, const double* const f[8]) {
    for (int i = 0; i < 8; ++i) if (!f[i]) return c->fail(MHD_ERR_INVALID_ARG, "null field pointer");
    SlabIO io; io.nin = 0; io.nout = 8; io.kind = kind; io.where = where; io.user_in = f;
    int rc = stage_slabs(c, SLAB_FROM_REAL, io);
    if (rc) return rc;
    if (c->ooc.world > 1) {            // exchange, then MHD_DIST_PHASE_STORE
        if (where == MHD_HOST) cudaStreamSynchronize(c->st);     // the caller's host buffers are free again on return
        return check_cuda(c, "set_fields (decomposed, slab part)");
    }
    rc = stage_forward_z_store(c);
    if (rc) return rc;
    if (where == MHD_HOST) cudaStreamSynchronize(c->st);
    return check_cuda(c, "set_fields (chunked)");
}

int ooc_get_fields(mhd_ctx* c, int kind, int where, double* const out[8]) {
    for (int i = 0; i < 8; ++i) if (!out[i]) return c->fail(MHD_ERR_INVALID_ARG, "null field pointer");
    int rc = c->ooc.world > 1 ? MHD_OK : stage_inverse_z(c, c->ooc.Uc, false);   // decomposed: MHD_DIST_PHASE_STATE_Z + exchange came first
    if (rc) return rc;
    SlabIO io; io.nin = 8; io.nout = 0; io.kind = kind; io.where = where; io.user_out = out;
    rc = stage_slabs(c, SLAB_TO_REAL, io);
    if (rc) return rc;
    if (where == MHD_HOST) cudaStreamSynchronize(c->st);
    return check_cuda(c, "get_fields (chunked)");
}

// real-space conservative fields of the current state into DEVICE arrays; out[f] == null: field f is not wanted
// (tracers: B for the push, rho and m for the initial velocity)
int ooc_real_fields(mhd_ctx* c, double* const out[8]) {
    if (c->ooc.world > 1) return c->fail(MHD_ERR_INVALID_ARG, "not available on a decomposed context");
    int rc = stage_inverse_z(c, c->ooc.Uc, false);
    if (rc) return rc;
    SlabIO io; io.nin = 8; io.nout = 0; io.kind = MHD_CONSERVATIVE; io.where = MHD_DEVICE; io.user_out = out;
    rc = stage_slabs(c, SLAB_TO_REAL, io);
    return rc ? rc : check_cuda(c, "real fields (chunked)");
}

static int ooc_products(mhd_ctx* c, bool have_inverse_z = false) {
    if (!have_inverse_z) {
        int rc = stage_inverse_z(c, c->ooc.Uc, true);
        if (rc) return rc;
    }
    SlabIO io; io.nin = 11; io.nout = 16;
    return stage_slabs(c, SLAB_FLUX, io);
}

// the chunked pipeline implements the base equation set only: re-checked where the work is done, because the options can
// be set before mhd_bind makes the context a chunked one
static int ooc_variant_check(mhd_ctx* c) {
    if (c->f0 != 0.0) return c->fail(MHD_ERR_INVALID_ARG, "forcing (MHD_PARAM_FORCE_AMP) needs an in-core context");
    if (c->opt_stress) return c->fail(MHD_ERR_INVALID_ARG, "the stress-tensor variant (MHD_OPT_STRESS) needs an in-core context");
    return MHD_OK;
}

int ooc_rhs(mhd_ctx* c, int where, double* const out[8]) {
    if (int vrc = ooc_variant_check(c)) return vrc;
    if (c->ooc.world > 1) return c->fail(MHD_ERR_INVALID_ARG, "mhd_rhs is not available on a decomposed context");
    for (int i = 0; i < 8; ++i) if (!out[i]) return c->fail(MHD_ERR_INVALID_ARG, "null field pointer");
    int rc = ooc_products(c);
    if (rc) return rc;
    rc = stage_forward_z_assemble(c, 0, false);
    if (rc) return rc;
    SlabIO io; io.nin = 8; io.nout = 0; io.kind = MHD_CONSERVATIVE; io.where = where; io.user_out = out;
    rc = stage_slabs(c, SLAB_TO_REAL, io);
    if (rc) return rc;
    if (where == MHD_HOST) cudaStreamSynchronize(c->st);
    return check_cuda(c, "rhs (chunked)");
}

int ooc_step(mhd_ctx* c, int nsteps) {
    if (c->ooc.world > 1) return c->fail(MHD_ERR_INVALID_ARG, "decomposed context: drive the step with mhd_dist_phase and the exchanges");
    if (c->integrator != 0 && !c->ooc.stage_storage)
        return c->fail(MHD_ERR_INVALID_ARG, "RK4 / predictor-corrector on the chunked pipeline need MHD_FLAG_STAGE_STORAGE at mhd_bind");
    if (int vrc = ooc_variant_check(c)) return vrc;
    bool have_inverse_z = false;        // stage A of the next right-hand side already ran on the bricks of the last stage C
    for (int s = 0; s < nsteps; ++s) {
        if (c->integrator == 0) {
            int rc = ooc_products(c, have_inverse_z);
            if (rc) return rc;
            have_inverse_z = s + 1 < nsteps;
            rc = stage_forward_z_assemble(c, c->have_old ? 2 : 1, have_inverse_z);
            if (rc) return rc;
            c->have_old = true;
        } else {                        // RK4 / predictor-corrector, low-storage stages (kernels.h StageUpdate; mhd_api.cu mhd_step)
            const double dt = c->dt;
            const double rk4[4][2] = {{0.5 * dt, dt / 6.0}, {0.5 * dt, dt / 3.0}, {dt, dt / 3.0}, {0.0, dt / 6.0}};
            const double heun[2][2] = {{dt, 0.5 * dt}, {0.0, 0.5 * dt}};
            const int ns = c->integrator == 1 ? 4 : 2;
            for (int k = 0; k < ns; ++k) {
                StageUpdate sg = StageUpdate();
                sg.c_next = c->integrator == 1 ? rk4[k][0] : heun[k][0];
                sg.b_acc = c->integrator == 1 ? rk4[k][1] : heun[k][1];
                sg.first = k == 0; sg.last = k == ns - 1;
                int rc = ooc_products(c, have_inverse_z);
                if (rc) return rc;
                have_inverse_z = !(sg.last && s + 1 == nsteps);
                rc = stage_forward_z_assemble(c, 3, have_inverse_z, &sg);
                if (rc) return rc;
            }
            c->have_old = false;        // the R^old arrays now hold U0, not a slope
        }
        ++c->step;
    }
    return check_cuda(c, "step (chunked)");
}

int ooc_diagnostics(mhd_ctx* c, mhd_diag* d, double* spec_kin, double* spec_mag, int nspec) {
    Ooc& o = c->ooc;
    const int ns = nspec_of(c->N);
    if (o.world > 1) return c->fail(MHD_ERR_INVALID_ARG, "mhd_diagnostics is not available on a decomposed context");
    if (spec_kin) return c->fail(MHD_ERR_INVALID_ARG, "the kinetic spectrum needs an unpruned transform: not available in the chunked pipeline");
    if (spec_mag && nspec != ns) return c->fail(MHD_ERR_INVALID_ARG, "nspec must equal mhd_nspec(N)");
    int rc = stage_diag_bricks(c, spec_mag != nullptr);
    if (rc) return rc;
    SlabIO io; io.nin = 9; io.nout = 0; io.diag = true;
    rc = stage_slabs(c, SLAB_TO_REAL, io);
    if (rc) return rc;
    {
        mhd_ctx::Scope s(c, F_DIAG, 3);
        launch_diag_final(o.part_diag, c->res, 1.0 / (double)c->n3(), c->st);
        launch_absmax_final(o.part_max, c->res + 16, c->st);
        if (spec_mag) launch_shell_spectrum_final(o.part_spec, c->res + 64 + ns, ns, c->st);
    }
    std::vector<double> host(64 + 2 * ns);
    cudaMemcpyAsync(host.data(), c->res, host.size() * sizeof(double), cudaMemcpyDeviceToHost, c->st);
    cudaStreamSynchronize(c->st);
    rc = check_cuda(c, "diagnostics (chunked)");
    if (rc) return rc;
    d->t = (double)c->step * c->dt; d->step = c->step;
    d->ke = host[0]; d->me = host[1]; d->ie = host[2]; d->mass = host[3];
    d->mom[0] = host[4]; d->mom[1] = host[5]; d->mom[2] = host[6]; d->etot = host[7];
    d->rho_min = host[8]; d->p_min = host[9]; d->max_divb = host[16];
    if (spec_mag) std::memcpy(spec_mag, host.data() + 64 + ns, ns * sizeof(double));
    return MHD_OK;
}

// ---- slab decomposition over several GPUs (include/mhd.h mhd_dist_*) ------------------------------
// The chunked pipeline already separates what is local to a ky range (stages A, C: z passes, assembly, update) from what
// is local to a z range (stage B: y passes, fused x sweep).  Rank r of `world` runs A / C on its share of the compact ky
// axis and B on its share of the z planes; between them the z-full work arrays [z][ky_c][kx_c] are transposed across
// ranks by an all-to-all that the caller performs (torch.distributed / NCCL) on buffers packed and unpacked here.
int ooc_dist_config(mhd_ctx* c, int rank, int world) {
    Ooc& o = c->ooc;
    if (!o.on || o.state_host || o.work_host) return c->fail(MHD_ERR_INVALID_ARG, "decomposition needs MHD_FLAG_OUT_OF_CORE with everything in device memory");
    if (world < 1 || rank < 0 || rank >= world || world > o.nyc || world > c->N) return c->fail(MHD_ERR_INVALID_ARG, "rank / world");
    if (o.split && world != o.world) return c->fail(MHD_ERR_INVALID_ARG, "world must equal the MHD_FLAG_RANKS the context was bound with");
    o.rank = rank; o.world = world;
    c->have_fields = false; c->have_old = false; c->step = 0;
    return MHD_OK;
}

int ooc_dist_peers(mhd_ctx* c, const long long* delta_bytes) {
    Ooc& o = c->ooc;
    if (!o.on || o.world > 8) return c->fail(MHD_ERR_INVALID_ARG, "direct exchange: decomposed context with at most 8 ranks");
    o.direct = delta_bytes != nullptr;
    for (int s = 0; s < 8; ++s) o.peer_delta[s] = 0;
    if (delta_bytes)
        for (int s = 0; s < o.world; ++s) {
            if (delta_bytes[s] % (long long)sizeof(cd)) return c->fail(MHD_ERR_INVALID_ARG, "peer workspaces must be 16-byte congruent");
            o.peer_delta[s] = s == o.rank ? 0 : delta_bytes[s] / (long long)sizeof(cd);
        }
    return MHD_OK;
}

static int dist_phase_body(mhd_ctx* c, int phase, int arg);
int ooc_dist_phase(mhd_ctx* c, int phase, int arg) {
    Ooc& o = c->ooc;
    // rows go straight to their owners only in the phases of the step; set / get_fields use the packed exchange
    o.direct_active = o.direct && (phase == MHD_DIST_PHASE_A || phase == MHD_DIST_PHASE_B || phase == MHD_DIST_PHASE_C);
    const int rc = dist_phase_body(c, phase, arg);
    o.direct_active = false;
    return rc;
}
static int dist_phase_body(mhd_ctx* c, int phase, int arg) {
    switch (phase) {
        case MHD_DIST_PHASE_A: return stage_inverse_z(c, c->ooc.Uc, true);
        case MHD_DIST_PHASE_B: { SlabIO io; io.nin = 11; io.nout = 16; return stage_slabs(c, SLAB_FLUX, io); }
        case MHD_DIST_PHASE_C: {
            if (c->integrator != 0) return c->fail(MHD_ERR_INVALID_ARG, "the chunked pipeline implements Adams-Bashforth only");
            if (int vrc = ooc_variant_check(c)) return vrc;
            int rc = stage_forward_z_assemble(c, c->have_old ? 2 : 1, arg != 0);
            if (rc) return rc;
            c->have_old = true; ++c->step;
            return MHD_OK;
        }
        case MHD_DIST_PHASE_STORE: {
            int rc = stage_forward_z_store(c);
            if (rc) return rc;
            c->have_fields = true; c->have_old = false; c->step = 0;
            return MHD_OK;
        }
        case MHD_DIST_PHASE_STATE_Z: return stage_inverse_z(c, c->ooc.Uc, false);
        default: return c->fail(MHD_ERR_INVALID_ARG, "unknown phase");
    }
}

// block exchanged with peer s, in doubles.  dir 0 (bricks -> slabs): send my ky range x peer's z range, receive the peer's
// ky range x my z range; dir 1 (slabs -> bricks) the other way round.
int ooc_dist_counts(mhd_ctx* c, int dir, int nf, long long* send, long long* recv) {
    const Ooc& o = c->ooc;
    if ((dir != 0 && dir != 1) || nf < 1 || nf > 16) return c->fail(MHD_ERR_INVALID_ARG, "dir / nf");
    const long long ny_me = o.ky_lo(o.rank + 1) - o.ky_lo(o.rank), nz_me = o.z_lo(o.rank + 1, c->N) - o.z_lo(o.rank, c->N);
    for (int s = 0; s < o.world; ++s) {
        const long long ny_s = o.ky_lo(s + 1) - o.ky_lo(s), nz_s = o.z_lo(s + 1, c->N) - o.z_lo(s, c->N);
        long long a = 2LL * nf * nz_s * ny_me * o.nxp, b = 2LL * nf * nz_me * ny_s * o.nxp;
        if (s == o.rank) a = b = 0;          // the rank's own block (my ky range x my z range) is already in place
        if (send) send[s] = dir == 0 ? a : b;
        if (recv) recv[s] = dir == 0 ? b : a;
    }
    return MHD_OK;
}

// pack (unpack = 0): work arrays -> buf = [peer 0 block | peer 1 block | ...], block = [f][z][ky][kx_c]; unpack = 1: the
// received buffer of the same exchange -> work arrays.  One 2-D device copy per (peer, field) on the solver's stream.
int ooc_dist_pack(mhd_ctx* c, int dir, int nf, double* buf, int unpack) {
    const Ooc& o = c->ooc;
    if ((dir != 0 && dir != 1) || nf < 1 || nf > 16 || !buf) return c->fail(MHD_ERR_INVALID_ARG, "dir / nf / buffer");
    const int N = c->N, me = o.rank;
    cd* p = reinterpret_cast<cd*>(buf);
    const size_t plane = (size_t)o.nyc * o.nxp;
    for (int s = 0; s < o.world; ++s) {
        if (s == me) continue;                                   // own block: stays where it is
        // geometry of the block in the work arrays: which rank's z range and which rank's ky range
        const bool mine_ky = (dir == 0) != (unpack != 0);        // pack dir 0 / unpack dir 1: my ky, peer's z
        const int rz = mine_ky ? s : me, ry = mine_ky ? me : s;
        const int z0 = o.z_lo(rz, N), nz = o.z_lo(rz + 1, N) - z0, y0 = o.ky_lo(ry), ny = o.ky_lo(ry + 1) - y0;
        const size_t width = (size_t)ny * o.nxp;
        // "my ky, all z" lives in the brick-shaped arrays, "my z, all ky" in the slab-shaped ones (the same array when unified)
        const size_t pitch = mine_ky ? (size_t)o.bstride() : plane;
        for (int f = 0; f < nf; ++f) {
            cd* w = mine_ky ? o.WzB[f] + (size_t)z0 * pitch + (size_t)(y0 - o.yoff()) * o.nxp
                            : o.WzS[f] + (size_t)(z0 - o.zoff(N)) * pitch + (size_t)y0 * o.nxp;
            if (nz > 0 && ny > 0) {
                if (!unpack) cudaMemcpy2DAsync(p, width * sizeof(cd), w, pitch * sizeof(cd), width * sizeof(cd), nz, cudaMemcpyDeviceToDevice, c->st);
                else cudaMemcpy2DAsync(w, pitch * sizeof(cd), p, width * sizeof(cd), width * sizeof(cd), nz, cudaMemcpyDeviceToDevice, c->st);
            }
            p += width * nz;
        }
    }
    if (unpack && o.split) {
        // per-rank storage: the rank's own block (its ky share x its z share) changes arrays too — brick-shaped -> slab-shaped
        // for dir 0, the other way for dir 1 (with the unified layout both are the same memory and nothing moves)
        const int z0 = o.z_lo(me, N), nz = o.z_lo(me + 1, N) - z0, y0 = o.ky_lo(me), ny = o.ky_lo(me + 1) - y0;
        const size_t width = (size_t)ny * o.nxp, bp = (size_t)o.bstride();
        for (int f = 0; f < nf && nz > 0 && ny > 0; ++f) {
            cd* b = o.WzB[f] + (size_t)z0 * bp;                   // [z][ky - y0]
            cd* sl = o.WzS[f] + (size_t)y0 * o.nxp;               // [z - z0][ky]
            if (dir == 0) cudaMemcpy2DAsync(sl, plane * sizeof(cd), b, bp * sizeof(cd), width * sizeof(cd), nz, cudaMemcpyDeviceToDevice, c->st);
            else cudaMemcpy2DAsync(b, bp * sizeof(cd), sl, plane * sizeof(cd), width * sizeof(cd), nz, cudaMemcpyDeviceToDevice, c->st);
        }
    }
    return check_cuda(c, unpack ? "dist unpack" : "dist pack");
}

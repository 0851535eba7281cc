// tracers.cu — tracer particles of PAPER.md Sec. VI (L229-275): cloud-in-cell gather of the grid magnetic field
// (Eq. 20) + Boris rotation (Eq. 21) + position update with periodic wrap (Eq. 22), one thread per particle.
//
// The push is a pure gather: per particle 24 grid values (8 corners x 3 components) are read through the read-only
// path; the two x-neighbours of a corner pair share a 32-byte sector except at sector boundaries, so a particle
// touches ~12-16 sectors.  Particles are independent, so `nsteps` pushes in a frozen field run inside one launch.
// Roofline: HBM / L2 gather (sectors, not flops): ~150 fp64 operations against >= 384 B of sector traffic per push.
// Arithmetic follows the paper's order (readings T1-T4): cell index floor(x N/L) in fp64, weights = opposite
// sub-cell volumes, t = B dt/2, s = 2t/(1+t^2), v_d = v + v x t, v+ = v + v_d x s, x+ = x + v+ dt wrapped to [0, L).
#include "ctx.h"

namespace mhd {

namespace {

struct CellIdx {
    int i0[3], i1[3];
    double f[3];
};

__device__ __forceinline__ CellIdx locate(int N, double inv_dx, double x, double y, double z) {
    CellIdx c;
    const double p[3] = {x, y, z};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double s = p[a] * inv_dx;
        const double fl = floor(s);
        c.f[a] = s - fl;
        long long i = (long long)fl % N;
        if (i < 0) i += N;
        c.i0[a] = (int)i;
        c.i1[a] = (int)((i + 1) % N);
    }
    return c;
}

// Eq. 20 for one grid field
__device__ __forceinline__ double cic(const double* __restrict__ g, int N, const CellIdx& c) {
    const double fx = c.f[0], fy = c.f[1], fz = c.f[2];
    const long long z0 = (long long)c.i0[2] * N, z1 = (long long)c.i1[2] * N;
    const long long r00 = (z0 + c.i0[1]) * N, r10 = (z0 + c.i1[1]) * N, r01 = (z1 + c.i0[1]) * N, r11 = (z1 + c.i1[1]) * N;
    const double g000 = __ldg(g + r00 + c.i0[0]), g100 = __ldg(g + r00 + c.i1[0]);
    const double g010 = __ldg(g + r10 + c.i0[0]), g110 = __ldg(g + r10 + c.i1[0]);
    const double g001 = __ldg(g + r01 + c.i0[0]), g101 = __ldg(g + r01 + c.i1[0]);
    const double g011 = __ldg(g + r11 + c.i0[0]), g111 = __ldg(g + r11 + c.i1[0]);
    const double ax = 1.0 - fx, ay = 1.0 - fy, az = 1.0 - fz;
    double b = g000 * (ax * ay * az);
    b += g100 * (fx * ay * az);
    b += g010 * (ax * fy * az);
    b += g110 * (fx * fy * az);
    b += g001 * (ax * ay * fz);
    b += g101 * (fx * ay * fz);
    b += g011 * (ax * fy * fz);
    b += g111 * (fx * fy * fz);
    return b;
}

__device__ __forceinline__ double wrap(double x, double L) {
    x -= L * floor(x / L);
    if (x >= L) x -= L;
    if (x < 0.0) x = 0.0;
    return x;
}

__global__ void __launch_bounds__(128) tracer_push_kernel(const __grid_constant__ TracerArgs a) {
    const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= a.np) return;
    const int N = a.N;
    const double inv_dx = (double)N / a.L, dt = a.dt, L = a.L;
    double x = a.pos[0][m], y = a.pos[1][m], z = a.pos[2][m];
    double vx = a.vel[0][m], vy = a.vel[1][m], vz = a.vel[2][m];
    for (int s = 0; s < a.nsteps; ++s) {
        const CellIdx c = locate(N, inv_dx, x, y, z);
        const double bx = cic(a.B[0], N, c), by = cic(a.B[1], N, c), bz = cic(a.B[2], N, c);
        const double tx = bx * (dt / 2.0), ty = by * (dt / 2.0), tz = bz * (dt / 2.0);
        const double t2 = tx * tx + ty * ty + tz * tz;
        const double sx = 2.0 * tx / (1.0 + t2), sy = 2.0 * ty / (1.0 + t2), sz = 2.0 * tz / (1.0 + t2);
        const double dx_ = vx + (vy * tz - vz * ty), dy_ = vy + (vz * tx - vx * tz), dz_ = vz + (vx * ty - vy * tx);
        const double nx = vx + (dy_ * sz - dz_ * sy), ny = vy + (dz_ * sx - dx_ * sz), nz = vz + (dx_ * sy - dy_ * sx);
        vx = nx; vy = ny; vz = nz;
        x = wrap(x + vx * dt, L); y = wrap(y + vy * dt, L); z = wrap(z + vz * dt, L);
    }
    a.pos[0][m] = x; a.pos[1][m] = y; a.pos[2][m] = z;
    a.vel[0][m] = vx; a.vel[1][m] = vy; a.vel[2][m] = vz;
}

struct InitArgs { const double* rho; const double* m[3]; };

// v <- CIC of u = m/rho (the quotient is taken at the grid points, then interpolated: reading T3)
__global__ void __launch_bounds__(128) tracer_init_velocity_kernel(const __grid_constant__ TracerArgs a,
                                                                   const __grid_constant__ InitArgs g) {
    const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= a.np) return;
    const int N = a.N;
    const CellIdx c = locate(N, (double)N / a.L, a.pos[0][m], a.pos[1][m], a.pos[2][m]);
    const double fx = c.f[0], fy = c.f[1], fz = c.f[2];
    double v[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int k = 0; k < 8; ++k) {                     // same corner order as Eq. 20: x fastest, then y, then z
        const int ix = (k & 1) ? c.i1[0] : c.i0[0], iy = (k & 2) ? c.i1[1] : c.i0[1], iz = (k & 4) ? c.i1[2] : c.i0[2];
        const double w = ((k & 1) ? fx : 1.0 - fx) * ((k & 2) ? fy : 1.0 - fy) * ((k & 4) ? fz : 1.0 - fz);
        const long long i = ((long long)iz * N + iy) * N + ix;
        const double rho = __ldg(g.rho + i);
#pragma unroll
        for (int d = 0; d < 3; ++d) v[d] += (__ldg(g.m[d] + i) / rho) * w;
    }
#pragma unroll
    for (int d = 0; d < 3; ++d) a.vel[d][m] = v[d];
}

__global__ void tracer_wrap_kernel(const __grid_constant__ TracerArgs a) {
    const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= a.np) return;
#pragma unroll
    for (int d = 0; d < 3; ++d) a.pos[d][m] = wrap(a.pos[d][m], a.L);
}

unsigned blocks_for(long long np) { return (unsigned)((np + 127) / 128); }

// ---- spatial sort (counting sort by grid row) ------------------------------------------------------------------
// Random particle order makes the gather DRAM-bound at sector granularity (ncu: ~670 B of DRAM reads per push at 256^3,
// against 48 B of particle state).  Sorted by the (z, y) row of their cell, consecutive threads read the same few grid
// rows, which then come from L1 / L2.  key = (iz * N + iy) * xb + coarse x (<= 2^20 bins); three kernels: histogram (the atomic's
// return value is the particle's rank inside its bin), exclusive scan of the bins, scatter.  The order inside a bin
// depends on the atomics, but every particle's own trajectory does not depend on where it is stored, and
// mhd_tracers_get un-permutes by id: results are bitwise independent of the sort.
__host__ __device__ inline unsigned sort_xbins(int N) {
    const unsigned cap = (1u << 20) / ((unsigned)N * (unsigned)N);
    return cap >= 16 ? 16u : (cap >= 4 ? 4u : 1u);
}
__global__ void sort_hist_kernel(const __grid_constant__ TracerArgs a, unsigned* __restrict__ hist, unsigned* __restrict__ key,
                                 unsigned* __restrict__ rank) {
    const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= a.np) return;
    const CellIdx c = locate(a.N, (double)a.N / a.L, a.pos[0][m], a.pos[1][m], a.pos[2][m]);
    // (z, y) row of the cell, refined by a coarse x index while the bins fit (xb = 1, 4, 16 sub-bins per row at 1024, 512, <= 256)
    const unsigned xb = sort_xbins(a.N);
    const unsigned k = ((unsigned)c.i0[2] * (unsigned)a.N + (unsigned)c.i0[1]) * xb + (unsigned)c.i0[0] * xb / (unsigned)a.N;
    key[m] = k;
    rank[m] = atomicAdd(&hist[k], 1u);
}
// exclusive scan of n <= 2^20 bins by one block of 1024 threads (each thread owns a contiguous run)
__global__ void __launch_bounds__(1024) sort_scan_kernel(unsigned* __restrict__ hist, int n) {
    __shared__ unsigned part[1024];
    const int t = threadIdx.x, per = (n + 1023) / 1024, lo = t * per, hi = min(n, lo + per);
    unsigned s = 0;
    for (int i = lo; i < hi; ++i) s += hist[i];
    part[t] = s;
    __syncthreads();
    for (int d = 1; d < 1024; d <<= 1) {
        const unsigned v = t >= d ? part[t - d] : 0u;
        __syncthreads();
        part[t] += v;
        __syncthreads();
    }
    unsigned run = part[t] - s;
    for (int i = lo; i < hi; ++i) { const unsigned h = hist[i]; hist[i] = run; run += h; }
}
struct SortIO { const double* src[6]; double* dst[6]; const long long* id_src; long long* id_dst; };
__global__ void sort_scatter_kernel(long long np, const unsigned* __restrict__ hist, const unsigned* __restrict__ key,
                                    const unsigned* __restrict__ rank, const __grid_constant__ SortIO io) {
    const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= np) return;
    const long long d = (long long)hist[key[m]] + rank[m];
#pragma unroll
    for (int f = 0; f < 6; ++f) io.dst[f][d] = io.src[f][m];
    io.id_dst[d] = io.id_src[m];
}
__global__ void iota_kernel(long long np, long long* id) {
    const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m < np) id[m] = m;
}
// out[id[m]] = in[m]
__global__ void unpermute_kernel(long long np, const long long* __restrict__ id, const double* __restrict__ in, double* __restrict__ out) {
    const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m < np) out[id[m]] = in[m];
}

}  // namespace

void launch_tracer_iota(long long np, long long* id, cudaStream_t st) {
    if (np > 0) iota_kernel<<<blocks_for(np), 128, 0, st>>>(np, id);
}
void launch_tracer_unpermute(long long np, const long long* id, const double* in, double* out, cudaStream_t st) {
    if (np > 0) unpermute_kernel<<<blocks_for(np), 128, 0, st>>>(np, id, in, out);
}
// sorts (pos, vel, id) into (alt_pos, alt_vel, alt_id); the caller swaps the buffers.  4 launches + one memset.
void launch_tracer_sort(const TracerArgs& a, const long long* id, double* const alt[6], long long* alt_id, unsigned* hist,
                        unsigned* key, unsigned* rank, cudaStream_t st) {
    if (a.np <= 0) return;
    const int nbins = a.N * a.N * (int)sort_xbins(a.N);
    cudaMemsetAsync(hist, 0, (size_t)nbins * sizeof(unsigned), st);
    sort_hist_kernel<<<blocks_for(a.np), 128, 0, st>>>(a, hist, key, rank);
    sort_scan_kernel<<<1, 1024, 0, st>>>(hist, nbins);
    SortIO io;
    for (int d = 0; d < 3; ++d) { io.src[d] = a.pos[d]; io.src[3 + d] = a.vel[d]; }
    for (int f = 0; f < 6; ++f) io.dst[f] = alt[f];
    io.id_src = id; io.id_dst = alt_id;
    sort_scatter_kernel<<<blocks_for(a.np), 128, 0, st>>>(a.np, hist, key, rank, io);
}

void launch_tracer_push(const TracerArgs& a, cudaStream_t st) {
    if (a.np > 0) tracer_push_kernel<<<blocks_for(a.np), 128, 0, st>>>(a);
}
void launch_tracer_init_velocity(const TracerArgs& a, const double* rho, const double* const m[3], cudaStream_t st) {
    InitArgs g{rho, {m[0], m[1], m[2]}};
    if (a.np > 0) tracer_init_velocity_kernel<<<blocks_for(a.np), 128, 0, st>>>(a, g);
}
void launch_tracer_wrap(const TracerArgs& a, cudaStream_t st) {
    if (a.np > 0) tracer_wrap_kernel<<<blocks_for(a.np), 128, 0, st>>>(a);
}

}  // namespace mhd

// kernels_strided.cu — complex fp64 FFT passes along the strided axes (y, z) of [kz][ky][kx] arrays.
//
// One CTA owns a tile of N rows (the transformed axis) x C consecutive kx columns (C*16 B = one 128-byte
// line per row for C = 8).  Each thread loads its E points straight into registers (16-byte loads, 8 lanes
// cover one full 128-byte line, 4 lines per warp instruction, E independent loads in flight per thread),
// the autosort exchange runs through a shared-memory tile [row][C] (conflict free, see fft_core.cuh), and
// the results go straight back to global memory in the same pattern — in place is safe because the tile
// is private to the CTA.  HBM-bound: 16 B read + 16 B written per point, one shared-memory round trip per
// stage boundary.  2/3-rule pruning: rows, columns and outer indices that the dealias mask makes
// identically zero are neither read nor written.
#include "fft_core.cuh"
#include "kernels.h"
#include "physics.cuh"

#include <cooperative_groups.h>
#include <cstdlib>
namespace cg = cooperative_groups;

namespace mhd {

// stored index of transform row `row` (mode 2 = compact, see kernels.h), or -1 if the row is not stored / not used
template <int N> __device__ __forceinline__ int stored_row(int row, int mode, int kc) {
    if (mode == 0) return row;
    if (row <= kc) return row;
    if (row >= N - kc) return mode == 2 ? row - (N - 2 * kc - 1) : row;
    return -1;
}

// GEN = false: the in-core sweeps (input and output views share their strides, rows stored in full: modes 0 / 1);
//               this is the tuned hot path, its address arithmetic folds to constants.
// GEN = true : bricks and slabs of the pipelined / out-of-core path (separate views, compact rows: any mode).
// FJ         : inverse z pass that builds J^ = M i k x B^ on load (sweep S1) for the fields f >= jfirst.
// at most 128 registers per thread, so that 512 threads (N = 512: two CTAs) stay resident per SM
template <int N, int C> struct StridedOcc {
    static constexpr int THREADS = C * PlanInfo<N>::T;
    static constexpr int MINB = (512 / THREADS) < 1 ? 1 : ((512 / THREADS) > 8 ? 8 : (512 / THREADS));
};
// line plan of the register-fed kernel: N = 512 with 8 columns uses the one-exchange plan (32 points per thread, radix 32 x 16,
// 128 threads and <= 168 registers: three 64 KB tiles per SM instead of two, one shared-memory round trip instead of two)
template <int N, int C> struct SPlan { typedef Plan<N> type; static constexpr int MINB = StridedOcc<N, C>::MINB; };
#ifndef MHD_STRIDED_512_TWO_EXCHANGES
template <> struct SPlan<512, 8> { typedef Plan512x type; static constexpr int MINB = 3; };
// (the same idea at N = 1024 — radix 32 x 32, 4-column tiles, three CTAs per SM — measured slower: 51.7 + 70.0 ms against
// 48.1 + 67.2 ms per step of the chunked pipeline; the twiddled radix-32 stage needs 16 table roots and spills)
#endif

template <int N, int DIR, int C, bool GEN, bool FJ>
__global__ void __launch_bounds__(C * (N / SPlan<N, C>::type::E), SPlan<N, C>::MINB)
strided_kernel(const __grid_constant__ StridedArgs a) {
    typedef typename SPlan<N, C>::type PL;
    constexpr int E = PL::E, T = N / PL::E;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* sm = reinterpret_cast<cd*>(smem_raw);

    const int tid = threadIdx.x;
    const int c = tid % C, t = tid / C;
    // FJ: the field is the fastest block index, so that the CTAs which read the same B^ tile (B itself and the two J
    // components built from it) run back to back and share it through L2 instead of fetching it from DRAM three times
    const int bx = FJ ? blockIdx.x / a.nfields : blockIdx.x;
    const int col = bx * C + c;
    int o = blockIdx.y;
    if (!GEN && o >= a.outer_split) o += a.outer_skip;
    const int f = FJ ? blockIdx.x % a.nfields : blockIdx.z;
    const bool valid = col < a.ncols;
    const int kc = a.kc;

    cd v[E];
    if (FJ && f >= a.jfirst) {
        // J^_c = M (i k x B^)_c built on load: rows are kz, the outer index is ky, columns are kx
        const int comp = f - a.jfirst;                       // 0: x, 1: y, 2: z
        const int ca = comp == 2 ? 0 : comp + 1, cb = comp == 0 ? 2 : comp - 1;   // J_c = i (k_ca B_cb - k_cb B_ca)
        const long long base = (long long)o * a.in_outer_stride + col;
        const cd* __restrict__ Ba = a.in[a.bfirst + ca] + base;
        const cd* __restrict__ Bb = a.in[a.bfirst + cb] + base;
        int ny;
        if (GEN && a.outer_compact) { const int oc = blockIdx.y + a.outer_base; ny = oc <= kc ? oc : oc - (2 * kc + 1); }
        else ny = o <= N / 2 ? o : o - N;
        const bool col_in = valid && col <= kc && abs(ny) <= kc;
        const double kxv = a.k0 * col, kyv = a.k0 * ny;
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const int row = t + T * m;
            const int nz = row <= N / 2 ? row : row - N;
            const int sr = GEN ? stored_row<N>(row, a.in_rows, kc) : row;
            cd ba = mk(0.0, 0.0), bb = ba;
            if (col_in && abs(nz) <= kc) { ba = Ba[(long long)sr * a.in_row_stride]; bb = Bb[(long long)sr * a.in_row_stride]; }
            const double kzv = a.k0 * nz;
            const double ka = ca == 0 ? kxv : (ca == 1 ? kyv : kzv), kb = cb == 0 ? kxv : (cb == 1 ? kyv : kzv);
            v[m] = mk(-(ka * bb.y) + kb * ba.y, ka * bb.x - kb * ba.x);      // i (ka bb - kb ba)
        }
    } else {
        const cd* __restrict__ in = a.in[f] + (long long)o * a.in_outer_stride + col;
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const int row = t + T * m;
            if (GEN) {
                const int sr = stored_row<N>(row, a.in_rows, kc);
                v[m] = (valid && sr >= 0) ? in[(long long)sr * a.in_row_stride] : mk(0.0, 0.0);
            } else {
                const bool keep = valid && (!a.in_rows || row <= kc || row >= N - kc);
                v[m] = keep ? in[(long long)row * a.in_row_stride] : mk(0.0, 0.0);
            }
        }
    }
    fft_line<N, DIR, 1, LayoutPlain, BlockSync, PL>(v, t, a.tw, sm, LayoutPlain{C, c});
    if (GEN) {
        cd* __restrict__ out = a.out[f] + (long long)o * a.out_outer_stride + col;
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const int sr = stored_row<N>(t + T * m, a.out_rows, kc);
            if (valid && sr >= 0) {
                long long d = 0;
                if (a.npeer > 0) {              // the row's owner: a peer's workspace (P2P store) or this one
                    int p = 0;
                    while (p + 1 < a.npeer && sr >= a.peer_lo[p + 1]) ++p;
                    d = a.peer_delta[p];
                }
                out[(long long)sr * a.out_row_stride + d] = v[m];
            }
        }
    } else {
        cd* __restrict__ out = a.out[f] + (long long)o * a.in_outer_stride + col;
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const int row = t + T * m;
            const bool keep = valid && (!a.out_rows || row <= kc || row >= N - kc);
            if (keep) out[(long long)row * a.in_row_stride] = v[m];
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// Sweep S5 in one launch: forward z pass (in-core, pruned) + assembly of R^ + explicit update (kernels.h AssembleTail).
// Grid: x = (kx tile) * 16 + field, y = ky (pruned list); thread-block CLUSTERS of 16 along x, so that the 16 CTAs that
// transform the 16 product fields of one (ky, kx tile) column are co-scheduled (hardware guarantee) and see each other's
// shared memory.  Each CTA transforms its field (rows = kz) and leaves the rows inside the mask in its own tile; after a
// cluster barrier every CTA assembles 1/16 of the rows, reading the 16 product values of a mode from the 16 tiles through
// distributed shared memory.  The transformed products never reach L2 or HBM: sweep S5 reads 16 + 8 + 8 and writes 8 + 8
// field sweeps, as SURVEY.md 8(d) counts it.
// ---------------------------------------------------------------------------------------------------------------------
// FPC = product fields per CTA (1 or 2) -> clusters of 16 / FPC CTAs.  Shared memory: the exchange tile [N][8] plus, for
// FPC = 2, one compact tile [2kc+1][8] that keeps the first field's rows while the second field is transformed.
template <int N, int FPC, int CC> struct S5Cfg {
    static constexpr int C = CC, NK = 2 * (N / 3) + 1, CL = P_NOUT / FPC;
    static constexpr int RPC = (NK + CL - 1) / CL;                  // kept rows assembled per CTA
    static constexpr size_t SMEM = (size_t(N) * C + size_t(FPC - 1) * NK * C) * sizeof(cd);
};

template <int N, int FPC, int CC>
__global__ void __launch_bounds__(CC * (N / SPlan<N, CC>::type::E), SPlan<N, CC>::MINB)
strided_assemble_kernel(const __grid_constant__ StridedArgs a, const __grid_constant__ AssembleTail z) {
    typedef S5Cfg<N, FPC, CC> P;
    typedef typename SPlan<N, CC>::type PL;      // same butterfly plan as the two-launch path: bitwise the same numbers
    constexpr int E = PL::E, T = N / PL::E, C = CC, NK = P::NK, CL = P::CL, RPC = P::RPC;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* sm = reinterpret_cast<cd*>(smem_raw);
    cg::cluster_group cluster = cg::this_cluster();

    const int tid = threadIdx.x;
    const int c = tid % C, t = tid / C;
    const int bx = blockIdx.x / CL, rank = blockIdx.x % CL;           // rank in the cluster
    const int col = bx * C + c;
    int o = blockIdx.y;
    if (o >= a.outer_split) o += a.outer_skip;
    const bool valid = col < a.ncols;
    const int kc = a.kc;
    const long long base = (long long)o * a.in_outer_stride + col;

    // the state lines this CTA will update after the barrier: start them on their way to L2 now
    if (c == 0 && bx * C <= kc) {
        for (int ri = t; ri < RPC; ri += T) {
            const int i = rank * RPC + ri;
            if (i >= NK) break;
            const int row = i <= kc ? i : i + (N - NK);
            const long long line = base + (long long)row * a.in_row_stride;
#pragma unroll
            for (int g = 0; g < 8; ++g) {
                asm volatile("prefetch.global.L2 [%0];" ::"l"(z.U[g] + line));
                if (z.mode == 2) asm volatile("prefetch.global.L2 [%0];" ::"l"(z.Rold[g] + line));
            }
        }
    }
#pragma unroll
    for (int fi = 0; fi < FPC; ++fi) {
        const int f = rank * FPC + fi;
        cd v[E];
        const cd* __restrict__ in = a.in[f] + base;
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = valid ? in[(long long)(t + T * m) * a.in_row_stride] : mk(0.0, 0.0);
        if (fi > 0) __syncthreads();        // the previous field's compact rows have left the exchange tile
        fft_line<N, -1, 1, LayoutPlain, BlockSync, PL>(v, t, a.tw, sm, LayoutPlain{C, c});
        __syncthreads();                    // every thread has gathered its last exchange: the tile is free
        // kept rows, compact index i: the last field of the CTA stays in the exchange tile, earlier ones move behind it
        cd* keep = (fi == FPC - 1) ? sm : sm + (size_t)N * C + (size_t)fi * NK * C;
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const int row = t + T * m;
            if (row <= kc) keep[row * C + c] = v[m];
            else if (row >= N - kc) keep[(row - (N - NK)) * C + c] = v[m];
        }
    }
    cluster.sync();                         // all 16 product tiles of this column are in place
    // ---- assembly: this CTA takes the kept rows [rank * RPC, (rank + 1) * RPC) --------------------------------------
    if (valid && col <= kc) {
        const int ny = o <= N / 2 ? o : o - N;
        const double kxv = z.ph.k0 * col, kyv = z.ph.k0 * ny;
        for (int ri = t; ri < RPC; ri += T) {
            const int i = rank * RPC + ri;
            if (i >= NK) break;
            const int row = i <= kc ? i : i + (N - NK);
            const int nz = row <= N / 2 ? row : row - N;
            const long long idx = base + (long long)row * a.in_row_stride;
            cd u[8], R[8];
#pragma unroll
            for (int g = 0; g < 8; ++g) u[g] = z.U[g][idx];
            auto ld = [&](int s) {
                const cd* tile = cluster.map_shared_rank(sm, s / FPC);
                const int fi = s % FPC;
                if (fi != FPC - 1) tile += (size_t)N * C + (size_t)fi * NK * C;
                return tile[i * C + c];
            };
            rhs_mode(ld, u, kxv, kyv, z.ph.k0 * nz, z.ph, R);
            if (z.mode == 0) {
#pragma unroll
                for (int g = 0; g < 8; ++g) z.rout[g][idx] = R[g];
            } else {
#pragma unroll
                for (int g = 0; g < 8; ++g) {
                    const cd ro = z.mode == 2 ? z.Rold[g][idx] : mk(0, 0);
                    z.U[g][idx] = updated(z.mode, z.dt, u[g], R[g], ro);
                    z.Rold[g][idx] = R[g];
                }
            }
        }
    }
    cluster.sync();                         // nobody leaves while its tile may still be read
}

template <int N, int FPC, int CC> static void s5_configure(cudaLaunchConfig_t& cfg, cudaLaunchAttribute* attr, const StridedArgs& a,
                                                   cudaStream_t st) {
    typedef S5Cfg<N, FPC, CC> P;
    configure_kernel(reinterpret_cast<const void*>(strided_assemble_kernel<N, FPC, CC>), P::SMEM, P::CL > 8);
    cfg = cudaLaunchConfig_t{};
    cfg.gridDim = dim3(((a.ncols + P::C - 1) / P::C) * P::CL, a.n_outer, 1);
    cfg.blockDim = dim3(P::C * (N / SPlan<N, CC>::type::E), 1, 1);
    cfg.dynamicSmemBytes = P::SMEM;
    cfg.stream = st;
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = P::CL; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
}
template <int N, int FPC, int CC> static void strided_assemble_one(const StridedArgs& a, const AssembleTail& z, cudaStream_t st) {
    cudaLaunchConfig_t cfg; cudaLaunchAttribute attr[1];
    s5_configure<N, FPC, CC>(cfg, attr, a, st);
    cudaLaunchKernelEx(&cfg, strided_assemble_kernel<N, FPC, CC>, a, z);
}
template <int N, int FPC, int CC> static int s5_max_clusters(const StridedArgs& a) {
    cudaLaunchConfig_t cfg; cudaLaunchAttribute attr[1];
    s5_configure<N, FPC, CC>(cfg, attr, a, nullptr);
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, strided_assemble_kernel<N, FPC, CC>, &cfg) != cudaSuccess) { cudaGetLastError(); return -1; }
    return n;
}
bool strided_assemble_supported(int N) { return N >= 64 && N <= 512; }
// variant: 1 = one field per CTA (clusters of 16); 2 = two fields per CTA (clusters of 8, the portable size)
void launch_strided_assemble(int N, int variant, const StridedArgs& a, const AssembleTail& z, cudaStream_t st) {
#define S5_CASE(NN)                                                             \
    case NN:                                                                    \
        if (variant == 1) strided_assemble_one<NN, 1, 8>(a, z, st);             \
        else strided_assemble_one<NN, 2, 8>(a, z, st);                          \
        break;
    switch (N) {
        S5_CASE(64) S5_CASE(128) S5_CASE(256) S5_CASE(512)
        default: break;
    }
#undef S5_CASE
}
int strided_assemble_max_clusters(int N, int variant, const StridedArgs& a) {
    switch (N * 4 + variant) {
        case 64 * 4 + 1: return s5_max_clusters<64, 1, 8>(a);
        case 64 * 4 + 2: return s5_max_clusters<64, 2, 8>(a);
        case 128 * 4 + 1: return s5_max_clusters<128, 1, 8>(a);
        case 128 * 4 + 2: return s5_max_clusters<128, 2, 8>(a);
        case 256 * 4 + 1: return s5_max_clusters<256, 1, 8>(a);
        case 256 * 4 + 2: return s5_max_clusters<256, 2, 8>(a);
        case 512 * 4 + 1: return s5_max_clusters<512, 1, 8>(a);
        case 512 * 4 + 2: return s5_max_clusters<512, 2, 8>(a);
        default: return -1;
    }
}

template <int N, int DIR, int C, bool GEN, bool FJ> static void launch_one(const StridedArgs& a, cudaStream_t st) {
    constexpr int threads = C * (N / SPlan<N, C>::type::E);
    constexpr size_t smem = size_t(N) * C * sizeof(cd);
    ensure_dynamic_smem(strided_kernel<N, DIR, C, GEN, FJ>, smem);
    dim3 grid((a.ncols + C - 1) / C, a.n_outer, a.nfields);
    if (FJ) grid = dim3(grid.x * a.nfields, a.n_outer, 1);
    strided_kernel<N, DIR, C, GEN, FJ><<<grid, threads, smem, st>>>(a);
}

template <int N, int C> static void launch_dir(int dir, const StridedArgs& a, cudaStream_t st) {
    const bool gen = a.general != 0, fj = a.jfirst >= 0 && dir > 0;
    if (dir < 0) { if (gen) launch_one<N, -1, C, true, false>(a, st); else launch_one<N, -1, C, false, false>(a, st); }
    else if (gen) { if (fj) launch_one<N, +1, C, true, true>(a, st); else launch_one<N, +1, C, true, false>(a, st); }
    else { if (fj) launch_one<N, +1, C, false, true>(a, st); else launch_one<N, +1, C, false, false>(a, st); }
}

int strided_cols(int N) { return N >= 1024 ? 4 : 8; }

void launch_strided(int N, int dir, const StridedArgs& a, cudaStream_t st) {
    switch (N) {
        case 16: launch_dir<16, 8>(dir, a, st); break;
        case 32: launch_dir<32, 8>(dir, a, st); break;
        case 64: launch_dir<64, 8>(dir, a, st); break;
        case 128: launch_dir<128, 8>(dir, a, st); break;
        case 256: launch_dir<256, 8>(dir, a, st); break;
        case 512: launch_dir<512, 8>(dir, a, st); break;
        case 1024:
            // measured at 1024^3 (chunked pipeline in HBM): the write-heavy inverse passes gain 13 % from 128-byte segments
            // (8 columns, one 128 KB tile per SM), the forward passes lose 2 %: 8 columns for the inverse, 4 for the forward
            if (dir > 0) launch_dir<1024, 8>(dir, a, st);
            else launch_dir<1024, 4>(dir, a, st);
            break;
        default: break;
    }
}

}  // namespace mhd

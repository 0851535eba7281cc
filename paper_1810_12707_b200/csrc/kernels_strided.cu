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

template <int N, int DIR, int C, bool GEN, bool FJ>
__global__ void __launch_bounds__(StridedOcc<N, C>::THREADS, StridedOcc<N, C>::MINB)
strided_kernel(const __grid_constant__ StridedArgs a) {
    constexpr int E = PlanInfo<N>::E, T = PlanInfo<N>::T;
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
    fft_line<N, DIR, 1>(v, t, a.tw, sm, LayoutPlain{C, c});
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

template <int N, int DIR, int C, bool GEN, bool FJ> static void launch_one(const StridedArgs& a, cudaStream_t st) {
    constexpr int threads = C * PlanInfo<N>::T;
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

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

template <int N, int DIR, int C>
__global__ void __launch_bounds__(C * PlanInfo<N>::T)
strided_kernel(const __grid_constant__ StridedArgs a) {
    constexpr int E = PlanInfo<N>::E, T = PlanInfo<N>::T;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* sm = reinterpret_cast<cd*>(smem_raw);

    const int tid = threadIdx.x;
    const int c = tid % C, t = tid / C;
    const int col = blockIdx.x * C + c;
    int o = blockIdx.y;
    if (o >= a.outer_split) o += a.outer_skip;
    const int f = blockIdx.z;
    const bool valid = col < a.ncols;
    const long long base = (long long)o * a.outer_stride + col;
    const cd* __restrict__ in = a.in[f] + base;
    cd* __restrict__ out = a.out[f] + base;
    const int kc = a.kc;

    cd v[E];
#pragma unroll
    for (int m = 0; m < E; ++m) {
        const int row = t + T * m;
        const bool keep = valid && (!a.in_pruned || row <= kc || row >= N - kc);
        v[m] = keep ? in[(long long)row * a.row_stride] : mk(0.0, 0.0);
    }
    fft_line<N, DIR, 1>(v, t, a.tw, sm, LayoutPlain{C, c});
#pragma unroll
    for (int m = 0; m < E; ++m) {
        const int row = t + T * m;
        const bool keep = valid && (!a.out_pruned || row <= kc || row >= N - kc);
        if (keep) out[(long long)row * a.row_stride] = v[m];
    }
}

template <int N, int DIR, int C> static void launch_one(const StridedArgs& a, cudaStream_t st) {
    constexpr int threads = C * PlanInfo<N>::T;
    constexpr size_t smem = size_t(N) * C * sizeof(cd);
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(strided_kernel<N, DIR, C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        configured = true;
    }
    dim3 grid(a.nchunks, a.n_outer, a.nfields);
    strided_kernel<N, DIR, C><<<grid, threads, smem, st>>>(a);
}

template <int N, int C> static void launch_dir(int dir, const StridedArgs& a, cudaStream_t st) {
    if (dir < 0) launch_one<N, -1, C>(a, st); else launch_one<N, +1, C>(a, st);
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
        case 1024: launch_dir<1024, 4>(dir, a, st); break;
        default: break;
    }
}

}  // namespace mhd

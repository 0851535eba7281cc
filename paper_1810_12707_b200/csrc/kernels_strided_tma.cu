// kernels_strided_tma.cu — the in-core strided (y / z) passes as a persistent, TMA-fed pipeline (north_star (1): "TMA-staged
// tile transposes for the strided axes"; PAPER.md L297-331 for the transforms, L351 "memory intensive").
//
// One CTA per SM walks over the tiles (N rows x 8 kx columns of one field) round-robin.  A ring of NBUF shared-memory
// tiles is filled by the tensor-memory accelerator — `cp.async.bulk.tensor` on a 4-D tensor map [field buffer][z][y][x]
// over the whole workspace, two boxes of rows per tile (pruned inputs: the rows inside the 2/3 mask only), completion
// counted in bytes on one mbarrier per ring slot — while G groups of warps, each with its own named barrier, transform
// the tiles that have landed: the loads of the next tiles are in flight during the whole transform of the current ones,
// so HBM never waits for a CTA to come back from its butterflies (the register-fed kernel of kernels_strided.cu has two
// tiles per SM which both load, then both compute).  The exchange of the autosort stages runs in place in the landed tile;
// when a group has gathered its last exchange the slot is handed back to the TMA for the tile NBUF positions ahead.
// Results leave through plain 16-byte stores (8 lanes = one 128-byte line), rows outside the mask are skipped.
//
// Shared memory: NBUF x N x 128 B = 192 KB (N = 512: 3 tiles, 2 groups of 256 threads; N = 256: 6 tiles, 4 groups of 128).
#include "fft_core.cuh"
#include "kernels.h"

#include <cuda.h>

#include <algorithm>
#include <cstddef>
#include <cstring>

namespace mhd {

namespace {

template <int N> struct TmaCfg {
    static constexpr int C = 8, T = PlanInfo<N>::T, E = PlanInfo<N>::E;
    static constexpr int GT = C * T;                 // threads of one group = one tile in flight through the butterflies
    static constexpr int G = 512 / GT;               // groups per CTA
    static constexpr int NBUF = G + G / 2;           // ring slots: G being transformed + G/2 landing
    static constexpr int TILE = N * C;               // complex elements per tile
    static constexpr size_t SMEM = size_t(NBUF) * TILE * sizeof(cd) + 256;   // + mbarriers + issue counters
    static_assert(G >= 2 && G <= 8, "group count");
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// one box of the 4-D tensor map -> shared memory; completes `bytes of the box` on the mbarrier
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* map, int c0, int c1, int c2, int c3, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}

struct TmaArgs {
    cd* out[MAXF];
    int fbuf[MAXF];        // field-buffer index (4th tensor coordinate) of each input array
    const cd* tw;
    long long row_stride, outer_stride;   // complex elements, of the output arrays (= the input arrays: in place or same shape)
    int nchunks, ncols, n_outer, outer_split, outer_skip, kc, in_rows, out_rows, nfields;
    int axis;              // 1: rows = y, outer = z;  2: rows = z, outer = ky
    int box_rows;          // rows per TMA box (two boxes per tile)
    long long ntiles;
};

template <int N, int DIR>
__global__ void __launch_bounds__(512, 1)
strided_tma_kernel(const __grid_constant__ CUtensorMap map, const __grid_constant__ TmaArgs a) {
    typedef TmaCfg<N> P;
    constexpr int C = P::C, T = P::T, E = P::E, GT = P::GT, G = P::G, NBUF = P::NBUF, TILE = P::TILE;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    cd* tiles = reinterpret_cast<cd*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + size_t(NBUF) * TILE * sizeof(cd));
    // issued[slot] = position (in this CTA's tile sequence) of the tile whose load was last issued into the slot
    volatile int* issued = reinterpret_cast<volatile int*>(smem_raw + size_t(NBUF) * TILE * sizeof(cd) + 128);

    const int tid = threadIdx.x, g = tid / GT, gt = tid % GT;
    const int c = gt % C, t = gt / C;
    const int kc = a.kc;
    const uint32_t tile_bytes = 2u * (uint32_t)a.box_rows * C * sizeof(cd);

    // tile w -> (kx chunk, outer index, field); the chunk is fastest so that concurrent CTAs touch neighbouring lines
    auto issue = [&](long long w, int slot) {
        const int bx = (int)(w % a.nchunks);
        const long long r = w / a.nchunks;
        int o = (int)(r % a.n_outer);
        const int f = (int)(r / a.n_outer);
        if (o >= a.outer_split) o += a.outer_skip;
        cd* dst = tiles + (size_t)slot * TILE;
        mbar_expect_tx(&full[slot], tile_bytes);
        const int r1 = N - a.box_rows;          // second box: the last box_rows rows (all rows: the second half)
        if (a.axis == 1) {
            tma_load_4d(dst, &map, bx * 2 * C, 0, o, a.fbuf[f], &full[slot]);
            tma_load_4d(dst + (size_t)r1 * C, &map, bx * 2 * C, r1, o, a.fbuf[f], &full[slot]);
        } else {
            tma_load_4d(dst, &map, bx * 2 * C, o, 0, a.fbuf[f], &full[slot]);
            tma_load_4d(dst + (size_t)r1 * C, &map, bx * 2 * C, o, r1, a.fbuf[f], &full[slot]);
        }
    };

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NBUF; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
#pragma unroll
        for (int s = 0; s < NBUF; ++s) {
            const long long w = (long long)blockIdx.x + (long long)s * gridDim.x;
            issued[s] = -1;
            if (w < a.ntiles) { issue(w, s); issued[s] = s; }
        }
    }
    __syncthreads();

    const GroupSync gsync{1 + g, GT};
    for (long long i = g;; i += G) {
        const long long w = (long long)blockIdx.x + i * gridDim.x;
        if (w >= a.ntiles) break;
        const int slot = (int)(i % NBUF);
        const uint32_t parity = (uint32_t)((i / NBUF) & 1);
        cd* sm = tiles + (size_t)slot * TILE;
        // try_wait tells phases apart by parity only: it must not start before the slot has been armed for THIS tile (else a
        // barrier that still waits for the tile NBUF positions back would read as complete).  The group that re-arms a slot
        // publishes the position it armed it for; the arming precedes the publication (fence), so once it is visible the
        // barrier is in this tile's phase or past it, and the parity wait is exact.
        while (issued[slot] < (int)i) { }
        mbar_wait(&full[slot], parity);

        const int bx = (int)(w % a.nchunks);
        const long long r = w / a.nchunks;
        int o = (int)(r % a.n_outer);
        const int f = (int)(r / a.n_outer);
        if (o >= a.outer_split) o += a.outer_skip;
        const int col = bx * C + c;
        const bool valid = col < a.ncols;

        cd v[E];
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const int row = t + T * m;
            const bool keep = !a.in_rows || row <= kc || row >= N - kc;
            v[m] = keep ? sm[row * C + c] : mk(0.0, 0.0);
        }
        gsync();                    // the tile has been read: it becomes the exchange buffer of the autosort stages
        fft_line<N, DIR, 1>(v, t, a.tw, sm, LayoutPlain{C, c}, gsync);
        gsync();                    // last exchange gathered by the whole group: the slot is free
        if (gt == 0) {
            const long long wn = (long long)blockIdx.x + (i + NBUF) * gridDim.x;
            if (wn < a.ntiles) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // our generic-proxy accesses before the TMA's writes
                issue(wn, slot);
                __threadfence_block();
                issued[slot] = (int)(i + NBUF);
            }
        }
        cd* __restrict__ out = a.out[f] + (long long)o * a.outer_stride + col;
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const int row = t + T * m;
            const bool keep = valid && (!a.out_rows || row <= kc || row >= N - kc);
            if (keep) out[(long long)row * a.row_stride] = v[m];
        }
    }
}

typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                             const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                             CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeFn encode_fn() {
    // a function-local static with an initialiser is set up exactly once, even when several host threads bind at once
    static const EncodeFn fn = [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            return reinterpret_cast<EncodeFn>(p);
        cudaGetLastError();
        return static_cast<EncodeFn>(nullptr);
    }();
    return fn;
}

template <int N, int DIR> void launch_tma_one(const CUtensorMap& map, const TmaArgs& a, int sms, cudaStream_t st) {
    typedef TmaCfg<N> P;
    ensure_dynamic_smem(strided_tma_kernel<N, DIR>, P::SMEM);
    const long long grid = std::min<long long>(a.ntiles, sms);
    strided_tma_kernel<N, DIR><<<(unsigned)grid, 512, P::SMEM, st>>>(map, a);
}

}  // namespace

bool strided_tma_supported(int N) { return N == 128 || N == 256 || N == 512; }

// Tensor maps over the field buffers of one workspace: base = first field buffer, `nbuf` buffers of `stride_bytes`, each an
// [N][N][N/2] complex = [N][N][N] double array.  maps[0]: rows = y, box rows = kc + 1; [1]: y, N/2; [2]: z, kc + 1; [3]: z, N/2.
bool strided_tma_build_maps(int N, void* base, size_t stride_bytes, int nbuf, void* maps_out /* 4 x CUtensorMap */) {
    EncodeFn enc = encode_fn();
    if (!enc || !strided_tma_supported(N)) return false;
    CUtensorMap* maps = static_cast<CUtensorMap*>(maps_out);
    const cuuint64_t dims[4] = {(cuuint64_t)N, (cuuint64_t)N, (cuuint64_t)N, (cuuint64_t)nbuf};
    const cuuint64_t strides[3] = {(cuuint64_t)N * 8, (cuuint64_t)N * N * 8, (cuuint64_t)stride_bytes};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    for (int m = 0; m < 4; ++m) {
        const cuuint32_t rows = (m & 1) ? N / 2 : N / 3 + 1;
        cuuint32_t box[4] = {16, 1, 1, 1};
        box[m < 2 ? 1 : 2] = rows;
        if (enc(&maps[m], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return false;
    }
    return true;
}

// true if the pass was launched; false: not eligible (the caller falls back to the register-fed kernel)
bool launch_strided_tma(int N, int dir, const StridedArgs& s, const StridedTma& tm, cudaStream_t st) {
    if (!tm.maps || !strided_tma_supported(N) || s.general || s.jfirst >= 0 || s.npeer > 0) return false;
    const long long hx = N / 2;
    int axis;
    if (s.in_row_stride == hx && s.in_outer_stride == (long long)N * hx) axis = 1;
    else if (s.in_row_stride == (long long)N * hx && s.in_outer_stride == hx) axis = 2;
    else return false;
    if (s.out_row_stride != s.in_row_stride || s.out_outer_stride != s.in_outer_stride) return false;
    TmaArgs a;
    std::memset(&a, 0, sizeof(a));
    for (int f = 0; f < s.nfields; ++f) {
        const ptrdiff_t d = reinterpret_cast<const char*>(s.in[f]) - static_cast<const char*>(tm.base);
        if (d < 0 || d % (ptrdiff_t)tm.stride_bytes != 0 || d / (ptrdiff_t)tm.stride_bytes >= tm.nbuf) return false;
        a.fbuf[f] = (int)(d / (ptrdiff_t)tm.stride_bytes);
        a.out[f] = s.out[f];
    }
    a.tw = s.tw; a.row_stride = s.in_row_stride; a.outer_stride = s.in_outer_stride;
    a.nchunks = (s.ncols + 7) / 8; a.ncols = s.ncols; a.n_outer = s.n_outer; a.outer_split = s.outer_split; a.outer_skip = s.outer_skip;
    a.kc = s.kc; a.in_rows = s.in_rows; a.out_rows = s.out_rows; a.nfields = s.nfields; a.axis = axis;
    a.box_rows = s.in_rows ? N / 3 + 1 : N / 2;
    a.ntiles = (long long)a.nchunks * a.n_outer * s.nfields;
    const CUtensorMap& map = static_cast<const CUtensorMap*>(tm.maps)[(axis == 1 ? 0 : 2) + (s.in_rows ? 0 : 1)];
    switch (N * 2 + (dir < 0 ? 0 : 1)) {
        case 128 * 2 + 0: launch_tma_one<128, -1>(map, a, tm.sms, st); break;
        case 128 * 2 + 1: launch_tma_one<128, +1>(map, a, tm.sms, st); break;
        case 256 * 2 + 0: launch_tma_one<256, -1>(map, a, tm.sms, st); break;
        case 256 * 2 + 1: launch_tma_one<256, +1>(map, a, tm.sms, st); break;
        case 512 * 2 + 0: launch_tma_one<512, -1>(map, a, tm.sms, st); break;
        case 512 * 2 + 1: launch_tma_one<512, +1>(map, a, tm.sms, st); break;
        default: return false;
    }
    return true;
}

}  // namespace mhd

// kernels_x.cu — passes along the contiguous (x, real) axis: R2C, C2R and the fused real-space sweep.
//
// A real line of N doubles is transformed as H = N/2 complex points z[n] = x[2n] + i x[2n+1] (the real array
// reinterpreted, no repacking) with the split/merge step fused into the load (C2R) or store (R2C):
//   R2C:  X[k] = (Z[k] + conj Z[H-k])/2 - (i/2) w^k (Z[k] - conj Z[H-k]),  w = exp(-2 pi i/N), k = 0..H-1
//   C2R:  Z'[k] = (X[k] + conj X[H-k]) + i conj(w^k) (X[k] - conj X[H-k]),  z = IFFT_H(Z')/N
// The Nyquist mode kx = N/2 is never stored: the 2/3 mask (R5) removes it from every quantity on
// the hot path, so half-spectrum rows are exactly H complex = N doubles, as long as the real rows
// (R2C can emit it to a side plane for the diagnostics spectra).
//
// SL lines share one CTA; the shared-memory tile is [n][SL] with the low 3 slot bits XOR-swizzled by the
// row so that both the coalesced global<->shared phases (lanes along n) and the FFT exchange phases (lanes
// along the slot) are bank-conflict free.
//
// x_fused_kernel is sweep S3 of the step: per (y,z) line it inverse-transforms the 11 fields
// (rho, m, E, B, J), forms the 16 flux products point-wise in shared memory and forward-transforms them,
// reading 11 and writing 16 half-spectrum lines: the real-space fields never touch HBM.
#include "fft_core.cuh"
#include "kernels.h"
#include "physics.cuh"

namespace mhd {

template <int SL> __device__ __forceinline__ int xidx(int n, int slot) { return n * SL + (slot ^ (n & 7)); }

// ---- C2R load: global half-spectrum lines -> Z' in the tile (pairs k, H-k) -----------------------------
template <int N, int SL>
__device__ __forceinline__ void c2r_load_pair(const cd* __restrict__ line, cd* sm, int slot, int k, int kmax,
                                              double scale, const cd* __restrict__ tw) {
    constexpr int H = N / 2;
    const cd zero = mk(0.0, 0.0);
    if (k == 0) {
        const cd x0 = line[0];
        const double a = scale * x0.x;              // the imaginary part of the mean mode carries no signal
        sm[xidx<SL>(0, slot)] = mk(a, a);
        const cd xh = (H / 2 <= kmax) ? line[H / 2] : zero;
        sm[xidx<SL>(H / 2, slot)] = mk(2.0 * scale * xh.x, -2.0 * scale * xh.y);
        return;
    }
    const cd A = (k <= kmax) ? line[k] : zero;
    const cd B = (H - k <= kmax) ? line[H - k] : zero;
    const cd w = __ldg(&tw[k]);
    const double Sx = A.x + B.x, Sy = A.y - B.y;     // S = A + conj(B)
    const double Dx = A.x - B.x, Dy = A.y + B.y;     // D = A - conj(B)
    const double p = w.x * Dx + w.y * Dy, q = w.x * Dy - w.y * Dx;
    sm[xidx<SL>(k, slot)] = mk(scale * (Sx - q), scale * (Sy + p));
    sm[xidx<SL>(H - k, slot)] = mk(scale * (Sx + q), scale * (p - Sy));
}

// ---- R2C store: Z in the tile -> global half-spectrum lines ---------------------------------------------
template <int N, int SL>
__device__ __forceinline__ void r2c_store_pair(cd* __restrict__ line, cd* __restrict__ nyq, const cd* sm, int slot,
                                               int k, int kmax, const cd* __restrict__ tw) {
    constexpr int H = N / 2;
    if (k == 0) {
        const cd z0 = sm[xidx<SL>(0, slot)];
        line[0] = mk(z0.x + z0.y, 0.0);
        if (nyq) nyq[0] = mk(z0.x - z0.y, 0.0);
        if (H / 2 <= kmax) {
            const cd zh = sm[xidx<SL>(H / 2, slot)];
            line[H / 2] = mk(zh.x, -zh.y);
        }
        return;
    }
    const cd Zk = sm[xidx<SL>(k, slot)], Zm = sm[xidx<SL>(H - k, slot)];
    const cd w = __ldg(&tw[k]);
    const double Sx = Zk.x + Zm.x, Sy = Zk.y - Zm.y;     // S = Zk + conj(Zm)
    const double Dx = Zk.x - Zm.x, Dy = Zk.y + Zm.y;     // D = Zk - conj(Zm)
    const double gx = w.x * Dx - w.y * Dy, gy = w.x * Dy + w.y * Dx;   // g = w D
    if (k <= kmax) line[k] = mk(0.5 * (Sx + gy), 0.5 * (Sy - gx));
    if (H - k <= kmax) line[H - k] = mk(0.5 * (Sx - gy), -0.5 * (Sy + gx));
}

// ---- H-point transform of the SL lines held in the tile, in place (natural order in and out) --------------
// nact: slots >= nact carry no data and skip the arithmetic (they still take part in the barriers)
template <int N, int SL, int DIR>
__device__ __forceinline__ void tile_fft(cd* sm, const cd* __restrict__ tw, int nact) {
    constexpr int H = N / 2, E = PlanInfo<H>::E, T = PlanInfo<H>::T;
    const int slot = threadIdx.x % SL, t = threadIdx.x / SL;
    const LayoutSwz L{SL, slot};
    cd v[E];
    const bool act = slot < nact;
    if (act) {
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = sm[L(t + T * m)];
    } else {
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = mk(0.0, 0.0);
    }
    __syncthreads();                           // tile free for the exchanges
    fft_line<H, DIR, 2>(v, t, tw, sm, L);
    __syncthreads();                           // last gather of every thread done
    if (act) {
#pragma unroll
        for (int m = 0; m < E; ++m) sm[L(t + T * m)] = v[m];
    }
    __syncthreads();
}

template <int N, int SL> struct XCfg {
    static constexpr int H = N / 2;
    static constexpr int T = PlanInfo<H>::T;
    static constexpr int THREADS = SL * T;
    static constexpr size_t SMEM = size_t(H) * SL * sizeof(cd);
};

// ---------------------------------------------------------------------------------------------------------
// generic R2C: grid (nlines/SL, nfields)
// ---------------------------------------------------------------------------------------------------------
template <int N, int SL>
__global__ void __launch_bounds__(XCfg<N, SL>::THREADS) x_r2c_kernel(const __grid_constant__ XArgs a) {
    constexpr int H = N / 2, NT = XCfg<N, SL>::THREADS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* sm = reinterpret_cast<cd*>(smem_raw);
    const int f = blockIdx.y;
    const long long line0 = (long long)blockIdx.x * SL;
    const double* __restrict__ rin = a.real_in[f];
    for (int i = threadIdx.x; i < SL * H; i += NT) {
        const int slot = i / H, n = i % H;
        sm[xidx<SL>(n, slot)] = reinterpret_cast<const cd*>(rin + (line0 + slot) * N)[n];
    }
    __syncthreads();
    tile_fft<N, SL, -1>(sm, a.tw, SL);
    cd* __restrict__ sout = a.spec_out[f];
    cd* __restrict__ nyq = a.nyq_out[f];
    for (int i = threadIdx.x; i < SL * (H / 2); i += NT) {
        const int slot = i / (H / 2), k = i % (H / 2);
        r2c_store_pair<N, SL>(sout + (line0 + slot) * H, nyq ? nyq + (line0 + slot) * 8 : nullptr, sm, slot, k,
                              a.kmax, a.tw);
    }
}

// ---------------------------------------------------------------------------------------------------------
// generic C2R: grid (nlines/SL, nfields)
// ---------------------------------------------------------------------------------------------------------
template <int N, int SL>
__global__ void __launch_bounds__(XCfg<N, SL>::THREADS) x_c2r_kernel(const __grid_constant__ XArgs a) {
    constexpr int H = N / 2, NT = XCfg<N, SL>::THREADS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* sm = reinterpret_cast<cd*>(smem_raw);
    const int f = blockIdx.y;
    const long long line0 = (long long)blockIdx.x * SL;
    const cd* __restrict__ sin_ = a.spec_in[f];
    for (int i = threadIdx.x; i < SL * (H / 2); i += NT) {
        const int slot = i / (H / 2), k = i % (H / 2);
        c2r_load_pair<N, SL>(sin_ + (line0 + slot) * H, sm, slot, k, a.kmax, a.scale, a.tw);
    }
    __syncthreads();
    tile_fft<N, SL, +1>(sm, a.tw, SL);
    double* __restrict__ rout = a.real_out[f];
    for (int i = threadIdx.x; i < SL * H; i += NT) {
        const int slot = i / H, n = i % H;
        reinterpret_cast<cd*>(rout + (line0 + slot) * N)[n] = sm[xidx<SL>(n, slot)];
    }
}

// ---------------------------------------------------------------------------------------------------------
// fused sweep S3: grid (nlines), one (y,z) line of all fields per CTA, SL = 16 slots
// ---------------------------------------------------------------------------------------------------------
template <int N>
__global__ void __launch_bounds__(XCfg<N, 16>::THREADS) x_fused_kernel(const __grid_constant__ FusedXArgs a) {
    constexpr int SL = 16, H = N / 2, NT = XCfg<N, SL>::THREADS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* sm = reinterpret_cast<cd*>(smem_raw);
    const long long off = (long long)blockIdx.x * H;

    for (int i = threadIdx.x; i < S_NIN * (H / 2); i += NT) {
        const int slot = i / (H / 2), k = i % (H / 2);
        c2r_load_pair<N, SL>(a.in[slot] + off, sm, slot, k, a.kmax_in, a.scale, a.tw);
    }
    __syncthreads();
    tile_fft<N, SL, +1>(sm, a.tw, S_NIN);

    // point-wise products: row n holds (f(x=2n), f(x=2n+1)) of every field
    for (int n = threadIdx.x; n < H; n += NT) {
        double s0[S_NIN], s1[S_NIN], o0[P_NOUT], o1[P_NOUT];
#pragma unroll
        for (int f = 0; f < S_NIN; ++f) {
            const cd z = sm[xidx<SL>(n, f)];
            s0[f] = z.x; s1[f] = z.y;
        }
        flux_point(s0, o0, a.ph);
        flux_point(s1, o1, a.ph);
#pragma unroll
        for (int f = 0; f < P_NOUT; ++f) sm[xidx<SL>(n, f)] = mk(o0[f], o1[f]);
    }
    __syncthreads();
    tile_fft<N, SL, -1>(sm, a.tw, P_NOUT);

    for (int i = threadIdx.x; i < P_NOUT * (H / 2); i += NT) {
        const int slot = i / (H / 2), k = i % (H / 2);
        r2c_store_pair<N, SL>(a.out[slot] + off, nullptr, sm, slot, k, a.kmax_out, a.tw);
    }
}

// ---------------------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------------------

template <int N> static void r2c_one(const XArgs& a, cudaStream_t st) {
    constexpr int SL = 8;
    ensure_dynamic_smem(x_r2c_kernel<N, SL>, XCfg<N, SL>::SMEM);
    dim3 grid((unsigned)(a.nlines / SL), a.nfields);
    x_r2c_kernel<N, SL><<<grid, XCfg<N, SL>::THREADS, XCfg<N, SL>::SMEM, st>>>(a);
}
template <int N> static void c2r_one(const XArgs& a, cudaStream_t st) {
    constexpr int SL = 8;
    ensure_dynamic_smem(x_c2r_kernel<N, SL>, XCfg<N, SL>::SMEM);
    dim3 grid((unsigned)(a.nlines / SL), a.nfields);
    x_c2r_kernel<N, SL><<<grid, XCfg<N, SL>::THREADS, XCfg<N, SL>::SMEM, st>>>(a);
}
template <int N> static void fused_one(const FusedXArgs& a, cudaStream_t st) {
    ensure_dynamic_smem(x_fused_kernel<N>, XCfg<N, 16>::SMEM);
    x_fused_kernel<N><<<(unsigned)a.nlines, XCfg<N, 16>::THREADS, XCfg<N, 16>::SMEM, st>>>(a);
}

#define MHD_DISPATCH_N(N, fn, ...)                  \
    switch (N) {                                    \
        case 16: fn<16>(__VA_ARGS__); break;        \
        case 32: fn<32>(__VA_ARGS__); break;        \
        case 64: fn<64>(__VA_ARGS__); break;        \
        case 128: fn<128>(__VA_ARGS__); break;      \
        case 256: fn<256>(__VA_ARGS__); break;      \
        case 512: fn<512>(__VA_ARGS__); break;      \
        case 1024: fn<1024>(__VA_ARGS__); break;    \
        default: break;                             \
    }

void launch_x_r2c(int N, const XArgs& a, cudaStream_t st) { MHD_DISPATCH_N(N, r2c_one, a, st) }
void launch_x_c2r(int N, const XArgs& a, cudaStream_t st) { MHD_DISPATCH_N(N, c2r_one, a, st) }
void launch_x_fused(int N, const FusedXArgs& a, cudaStream_t st) { MHD_DISPATCH_N(N, fused_one, a, st) }

}  // namespace mhd

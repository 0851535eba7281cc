// kernels_xfused2.cu — sweep S3, second generation: the fused real-axis kernel for N = 128, 256, 512, 1024.
//
// Per (y,z) line: C2R of 11 half-spectrum lines, 16 flux products, R2C of the 16 products.  Compared with the
// generic tile version (kernels_x.cu) this kernel
//   * maps lanes along the ROW index (t fastest): every quarter-warp reads / writes one full 128-byte line of one
//     field straight from / to global memory, E = 2*R0 independent 16-byte loads in flight per thread;
//   * folds the real-FFT split (C2R) and merge (R2C) into registers: the H-point transform is two stages
//     H = R0 x R1; thread t owns the first-stage butterflies j = t and j = R1 - t (t = 0: j = 0 and R1/2), whose
//     input rows j + r*R1 are exactly each other's mirror images k <-> H-k, so X[k], X[H-k] pairs meet in one thread;
//   * therefore moves 108 instead of 162 line-passes through shared memory per line (33 inverse, 27 point-wise,
//     48 forward) — shared-memory wavefronts were the largest term of the first version (ncu: profiles/);
//   * skips the arithmetic of the 5 idle slots of the inverse transform at warp granularity.
// The tile is [row][16 slots] with the slot XOR-swizzled by (row ^ row>>1 ^ row>>4) & 7, found by exhaustive search
// to make every scatter / gather / point-wise access of the H = 128 and H = 256 plans bank-conflict free.
#include "fft_core.cuh"
#include "kernels.h"
#include "physics.cuh"

#include <type_traits>

namespace mhd {

template <int H> struct FPlan;
template <> struct FPlan<64>  { static constexpr int R0 = 8,  R1 = 8;  };
template <> struct FPlan<128> { static constexpr int R0 = 8,  R1 = 16; };
template <> struct FPlan<256> { static constexpr int R0 = 16, R1 = 16; };
template <> struct FPlan<512> { static constexpr int R0 = 16, R1 = 32; };   // N = 1024: 128 KB tile, one CTA per SM

template <int H> struct F2 {
    static constexpr int R0 = FPlan<H>::R0, R1 = FPlan<H>::R1;
    static constexpr int T = R1 / 2;            // threads per slot
    static constexpr int NB = 2 * R0 / R1;      // radix-R1 butterflies per thread
    static constexpr int THREADS = 16 * T;
    static constexpr size_t SMEM = size_t(H) * 16 * sizeof(cd);
    static_assert(R0 * R1 == H, "two-stage plan");
};

template <int H> __device__ __forceinline__ int swz(int row) {
    if constexpr (H == 64) return (row ^ (row >> 1) ^ (row >> 2)) & 7;
    else return (row ^ (row >> 1) ^ (row >> 4)) & 7;
}
template <int H> __device__ __forceinline__ int tidx(int row, int slot) { return row * 16 + (slot ^ swz<H>(row)); }

// Lane-contiguous twiddle tables (built once at bind time, exact sincospi): consecutive lanes t read consecutive
// 16-byte entries, so one warp-wide twiddle load touches a single 128-byte line instead of up to 8 scattered ones
// (ncu on the first cut of this kernel: 3.4x more L1 load sectors than data because of scattered table reads).
//   TA[r][t] = exp(-2 pi i (jA(t) + r R1)/N)      split / merge factor of the rows of butterfly jA
//   TB[r][t] = exp(-2 pi i (jB(t) + r R1)/N)      same for butterfly jB (used by t = 0 only)
//   TS[b][e][t] = root e of the twiddle-folded radix-R1 butterfly j = t + b T of the second inverse stage
//                 (fft_core.cuh TDft: exp(-2 pi i 2^l (j + q R0)/H) for level l, position q)
//   TF[e][t]    = root e of the twiddle-folded radix-R0 butterfly jA = t of the last forward stage; the roots of its mirror
//                 butterfly jB = R1 - jA follow from them (mirror_roots); lane 0's jB = R1/2 has its own: TF[NR0 T + e]
template <int H> struct FTab {
    typedef F2<H> P;
    static constexpr int TA = 0;
    static constexpr int TB = P::R0 * P::T;
    static constexpr int TS = 2 * P::R0 * P::T;
    static constexpr int TF = TS + H;
    static constexpr int SIZE = TF + 2 * P::R0 * P::T;
};

// root e of TDft<R> for a butterfly with k = j mod Ns: exp(-2 pi i (2^l (k + q Ns)) / (Ns R)), (l, q) = position of e
__device__ inline void root_fraction(int R, int e, int k, int Ns, long long* num, int* den) {
    int Rl = R, l = 0;
    for (;;) {
        const int top = Rl >= 4 ? Rl / 4 : 1;
        if (e < top) break;
        e -= top; Rl /= 2; ++l;
    }
    *num = ((long long)k + (long long)e * Ns) << l;
    *den = Ns * R;
}
// roots of the mirror butterfly R1 - j (base exp(-2 pi i/R0) conj(w)) from those of butterfly j: level by level the entry
// a quarter turn away, conjugated and rotated — sign flips and swaps only
template <int R> __device__ __forceinline__ void mirror_roots(const cd* wa, cd* wb) {
    if constexpr (R >= 2) {
        constexpr int TOP = TwCount<R>::TOP;
        if constexpr (R >= 4) {
#pragma unroll
            for (int q = 0; q < TOP; ++q) { const cd a = wa[TOP - 1 - q]; wb[q] = mk(-a.y, -a.x); }
        } else {
            wb[0] = mk(-wa[0].x, wa[0].y);
        }
        mirror_roots<R / 2>(wa + TOP, wb + TOP);
    }
}

template <int H> __global__ void fused_twiddle_kernel(cd* tab) {
    typedef F2<H> P;
    constexpr int R0 = P::R0, R1 = P::R1, T = P::T, NB = P::NB, N = 2 * H;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= FTab<H>::SIZE) return;
    long long num; int den;
    if (i < FTab<H>::TS) {                       // TA, TB
        const int which = i / (R0 * T), r = (i % (R0 * T)) / T, t = i % T;
        const int j = which == 0 ? t : (t == 0 ? R1 / 2 : R1 - t);
        num = j + r * R1; den = N;
    } else if (i < FTab<H>::TF) {                // TS
        constexpr int NR1 = TwCount<R1>::value;
        const int k = i - FTab<H>::TS;
        if (k >= NB * NR1 * T) { tab[i] = mk(0.0, 0.0); return; }
        const int b = k / (NR1 * T), e = (k % (NR1 * T)) / T, t = k % T;
        root_fraction(R1, e, t + b * T, R0, &num, &den);
    } else {                                     // TF
        constexpr int NR0 = TwCount<R0>::value;
        const int k = i - FTab<H>::TF;
        if (k < NR0 * T) root_fraction(R0, k / T, k % T, R1, &num, &den);
        else if (k < NR0 * T + NR0) root_fraction(R0, k - NR0 * T, R1 / 2, R1, &num, &den);
        else { tab[i] = mk(0.0, 0.0); return; }
    }
    double sn, cs;
    sincospi(2.0 * (double)(num % den) / (double)den, &sn, &cs);
    tab[i] = mk(cs, -sn);
}

// compile-time loop: f(std::integral_constant<int, I>) for I = B .. E-1
template <int B, int E, class F> __device__ __forceinline__ void static_for(F&& f) {
    if constexpr (B < E) {
        f(std::integral_constant<int, B>{});
        static_for<B + 1, E>(f);
    }
}

// C2R split of one mirror pair: A = X[k], B = X[H-k], ws = scale * exp(-2 pi i k/N):  Z'[k] -> A, Z'[H-k] -> B, both
// scaled; the scale rides on the twiddle and on four FMAs (no separate multiplications)
__device__ __forceinline__ void c2r_pair(cd& A, cd& B, cd ws, double scale) {
    const double Sx = A.x + B.x, Sy = A.y - B.y;
    const double Dx = A.x - B.x, Dy = A.y + B.y;
    const double p = fma(ws.x, Dx, ws.y * Dy), q = fma(ws.x, Dy, -(ws.y * Dx));
    A = mk(fma(scale, Sx, -q), fma(scale, Sy, p));
    B = mk(fma(scale, Sx, q), fma(-scale, Sy, p));
}
// R2C merge of one mirror pair: Zk = Z[k], Zm = Z[H-k]:  X[k] -> Zk, X[H-k] -> Zm
// wh = w / 2: the halving rides on the twiddle and on four FMAs
__device__ __forceinline__ void r2c_pair(cd& Zk, cd& Zm, cd wh) {
    const double Sx = Zk.x + Zm.x, Sy = Zk.y - Zm.y;
    const double Dx = Zk.x - Zm.x, Dy = Zk.y + Zm.y;
    const double gx = fma(wh.x, Dx, -(wh.y * Dy)), gy = fma(wh.x, Dy, wh.y * Dx);
    Zk = mk(fma(0.5, Sx, gy), fma(0.5, Sy, -gx));
    Zm = mk(fma(0.5, Sx, -gy), fma(-0.5, Sy, -gx));
}

template <int N>
__global__ void __launch_bounds__(F2<N / 2>::THREADS, (N / 2 == 512) ? 1 : (N / 2 == 256) ? 3 : 5)
x_fused2_kernel(const __grid_constant__ FusedXArgs a) {
    constexpr int H = N / 2;
    typedef F2<H> P;
    constexpr int R0 = P::R0, R1 = P::R1, T = P::T, NB = P::NB, NT = P::THREADS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* sm = reinterpret_cast<cd*>(smem_raw);
    const cd* __restrict__ tab = a.tw;      // lane-contiguous tables (FTab)
    typedef FTab<H> FT;

    const int t = threadIdx.x % T, slot = threadIdx.x / T;
    const long long off = (long long)blockIdx.x * H;
    const int jA = t, jB = (t == 0) ? R1 / 2 : R1 - t;

    // ================= inverse: 11 lines, global -> registers -> tile =========================================
    if (slot < S_NIN) {
        const cd* __restrict__ line = a.in[slot] + off;
        const int kmax = a.kmax_in;
        const double scale = a.scale;
        cd xa[R0], xb[R0];
#pragma unroll
        for (int r = 0; r < R0; ++r) {
            const int ka = jA + r * R1, kb = jB + r * R1;
            xa[r] = (ka <= kmax) ? line[ka] : mk(0.0, 0.0);
            xb[r] = (kb <= kmax) ? line[kb] : mk(0.0, 0.0);
        }
        // split factors: exp(-2 pi i (j + r R1)/N) = exp(-2 pi i j/N) * (2 R0)-th root^r: one table load per thread
        if (t != 0) {
            const cd w0 = scale * __ldg(&tab[FT::TA + t]);
            static_for<0, R0>([&](auto rc) {
                constexpr int r = decltype(rc)::value;
                c2r_pair(xa[r], xb[R0 - 1 - r], mul_rootN<2 * R0, r, -1>(w0), scale);
            });
        } else {
            // rows r*R1: r = 0 is the mean mode (its mirror is the dropped Nyquist mode), r = R0/2 is k = H/2
            xa[0] = mk(scale * xa[0].x, scale * xa[0].x);
            xa[R0 / 2] = mk(2.0 * scale * xa[R0 / 2].x, -2.0 * scale * xa[R0 / 2].y);
            const cd one = mk(scale, 0.0);
            const cd wh = scale * __ldg(&tab[FT::TB]);  // scale * exp(-2 pi i (R1/2)/N)
            static_for<1, R0 / 2>([&](auto rc) {
                constexpr int r = decltype(rc)::value;
                c2r_pair(xa[r], xa[R0 - r], mul_rootN<2 * R0, r, -1>(one), scale);
            });
            static_for<0, R0 / 2>([&](auto rc) {
                constexpr int r = decltype(rc)::value;
                c2r_pair(xb[r], xb[R0 - 1 - r], mul_rootN<2 * R0, r, -1>(wh), scale);
            });
        }
        Dft<R0, +1>::run(xa);
        Dft<R0, +1>::run(xb);
#pragma unroll
        for (int q = 0; q < R0; ++q) {
            sm[tidx<H>(jA * R0 + q, slot)] = xa[q];
            sm[tidx<H>(jB * R0 + q, slot)] = xb[q];
        }
    }
    __syncwarp();           // a slot's T threads sit in one warp: its exchanges need no block-wide barrier
    if (slot < S_NIN) {
        // second stage: butterfly j reads and writes the same rows j + r*R0 -> in place, one butterfly at a time
#pragma unroll 1
        for (int b = 0; b < NB; ++b) {
            const int j = t + b * T;
            cd u[R1];
#pragma unroll
            for (int r = 0; r < R1; ++r) u[r] = sm[tidx<H>(j + r * R0, slot)];
            cd w[TwCount<R1>::value];
#pragma unroll
            for (int e = 0; e < TwCount<R1>::value; ++e) w[e] = __ldg(&tab[FT::TS + (b * TwCount<R1>::value + e) * T + t]);
            TDft<R1, +1>::run(u, w);
#pragma unroll
            for (int q = 0; q < R1; ++q) sm[tidx<H>(j + q * R0, slot)] = u[q];
        }
    }
    __syncthreads();        // the products read every slot of a row

    // ================= point-wise products: row n holds (f(x=2n), f(x=2n+1)) of every field ===================
#pragma unroll 1
    for (int n = threadIdx.x; n < H; n += NT) {
        double s0[S_NIN], s1[S_NIN], o0[P_NOUT], o1[P_NOUT];
#pragma unroll
        for (int f = 0; f < S_NIN; ++f) {
            const cd z = sm[tidx<H>(n, f)];
            s0[f] = z.x; s1[f] = z.y;
        }
        if (a.breal[0]) {           // tracers: the real-space B of this line also goes to HBM (block-uniform branch)
#pragma unroll
            for (int d = 0; d < 3; ++d)
                reinterpret_cast<cd*>(a.breal[d])[off + n] = mk(s0[S_BX + d], s1[S_BX + d]);
        }
        flux_point(s0, o0, a.ph);
        flux_point(s1, o1, a.ph);
#pragma unroll
        for (int f = 0; f < P_NOUT; ++f) sm[tidx<H>(n, f)] = mk(o0[f], o1[f]);
    }
    __syncthreads();

    // ================= forward: 16 lines, tile -> registers -> global ==========================================
    // first stage in place: Y[j][q] = sum_r x[j + r*R0] w_R1^(r q) is written back to row j + q*R0
#pragma unroll 1
    for (int b = 0; b < NB; ++b) {
        const int j = t + b * T;
        cd u[R1];
#pragma unroll
        for (int r = 0; r < R1; ++r) u[r] = sm[tidx<H>(j + r * R0, slot)];
        Dft<R1, -1>::run(u);
#pragma unroll
        for (int q = 0; q < R1; ++q) sm[tidx<H>(j + q * R0, slot)] = u[q];
    }
    __syncwarp();
    {
        cd* __restrict__ line = a.out[slot] + off;
        const int kmax = a.kmax_out;
        cd za[R0], zb[R0];
#pragma unroll
        for (int r = 0; r < R0; ++r) {
            za[r] = sm[tidx<H>(r + jA * R0, slot)];      // Y[r][jA]
            zb[r] = sm[tidx<H>(r + jB * R0, slot)];
        }
        // twiddle-folded butterflies: the roots of jA come from the table (lane 0: jA = 0, plain roots of unity), those of
        // jB = R1 - jA by mirror_roots; lane 0 (jB = R1/2) reads its own
        {
            constexpr int NR0 = TwCount<R0>::value;
            cd wa[NR0], wb[NR0];
#pragma unroll
            for (int e = 0; e < NR0; ++e) wa[e] = __ldg(&tab[FT::TF + e * T + t]);
            mirror_roots<R0>(wa, wb);
            if (t == 0) {
#pragma unroll
                for (int e = 0; e < NR0; ++e) wb[e] = __ldg(&tab[FT::TF + NR0 * T + e]);
            }
            TDft<R0, -1>::run(za, wa);
            TDft<R0, -1>::run(zb, wb);
        }
        // za[q] = Z[jA + q*R1], zb[q] = Z[jB + q*R1]
        if (t != 0) {
            const cd w0 = 0.5 * __ldg(&tab[FT::TA + t]);
            static_for<0, R0>([&](auto qc) {
                constexpr int q = decltype(qc)::value;
                r2c_pair(za[q], zb[R0 - 1 - q], mul_rootN<2 * R0, q, -1>(w0));
            });
        } else {
            za[0] = mk(za[0].x + za[0].y, 0.0);                         // k = 0 (Nyquist partner dropped)
            za[R0 / 2] = mk(za[R0 / 2].x, -za[R0 / 2].y);               // k = H/2
            const cd one = mk(0.5, 0.0);
            const cd wh = 0.5 * __ldg(&tab[FT::TB]);
            static_for<1, R0 / 2>([&](auto qc) {
                constexpr int q = decltype(qc)::value;
                r2c_pair(za[q], za[R0 - q], mul_rootN<2 * R0, q, -1>(one));
            });
            static_for<0, R0 / 2>([&](auto qc) {
                constexpr int q = decltype(qc)::value;
                r2c_pair(zb[q], zb[R0 - 1 - q], mul_rootN<2 * R0, q, -1>(wh));
            });
        }
#pragma unroll
        for (int q = 0; q < R0; ++q) {
            const int ka = jA + q * R1, kb = jB + q * R1;
            if (ka <= kmax) line[ka] = za[q];
            if (kb <= kmax) line[kb] = zb[q];
        }
    }
}

template <int N> static void fused2_one(const FusedXArgs& a, cudaStream_t st) {
    typedef F2<N / 2> P;
    ensure_dynamic_smem(x_fused2_kernel<N>, P::SMEM);
    x_fused2_kernel<N><<<(unsigned)a.nlines, P::THREADS, P::SMEM, st>>>(a);
}

bool x_fused2_supported(int N) { return N == 128 || N == 256 || N == 512 || N == 1024; }

int x_fused2_table_entries(int N) {
    switch (N) {
        case 128: return FTab<64>::SIZE;
        case 256: return FTab<128>::SIZE;
        case 512: return FTab<256>::SIZE;
        case 1024: return FTab<512>::SIZE;
        default: return 0;
    }
}
void launch_x_fused2_tables(int N, cd* tab, cudaStream_t st) {
    const int n = x_fused2_table_entries(N);
    if (n == 0) return;
    const int blocks = (n + 127) / 128;
    switch (N) {
        case 128: fused_twiddle_kernel<64><<<blocks, 128, 0, st>>>(tab); break;
        case 256: fused_twiddle_kernel<128><<<blocks, 128, 0, st>>>(tab); break;
        case 512: fused_twiddle_kernel<256><<<blocks, 128, 0, st>>>(tab); break;
        case 1024: fused_twiddle_kernel<512><<<blocks, 128, 0, st>>>(tab); break;
        default: break;
    }
}

void launch_x_fused2(int N, const FusedXArgs& a, cudaStream_t st) {
    switch (N) {
        case 128: fused2_one<128>(a, st); break;
        case 256: fused2_one<256>(a, st); break;
        case 512: fused2_one<512>(a, st); break;
        case 1024: fused2_one<1024>(a, st); break;
        default: break;
    }
}

}  // namespace mhd

// fft_core.cuh — register-resident fp64 Stockham FFT engine for sm_100a (device templates only).
//
// One "line" of NL complex points is transformed by T = NL/E threads, each holding E points in registers
// (v[m] <-> element t + T*m, the same ownership at entry and exit, so the first stage reads straight from
// global memory and the last stage writes straight to it).  Between stages the points are exchanged through
// a shared-memory tile whose fastest index is the line ("column"): 8 lanes with 8 different lines touch one
// 128-byte row, so every access pattern of the autosort exchange is bank-conflict free by construction.
// Stage s with radix R performs E/R butterflies per thread:
//     j = t + b*T,  k = j mod Ns,  u[r] = in[j + r*NL/R] * w^(r*k*NL/(Ns*R)),  u = DFT_R(u),
//     out[(j-k)*R + k + q*Ns] = u[q]                        (Ns = product of the radices already applied)
// which is the Stockham autosort formulation: natural order in, natural order out, no bit reversal.
// Twiddles come from an exactly rounded table w[m] = exp(-2*pi*i*m/NT) built once with sincospi (no
// recurrences: the fp64 error bound of the transform depends on it).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mhd {

typedef double2 cd;

__device__ __forceinline__ cd mk(double x, double y) { return make_double2(x, y); }
__device__ __forceinline__ cd operator+(cd a, cd b) { return mk(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cd operator-(cd a, cd b) { return mk(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cd operator*(double s, cd a) { return mk(s * a.x, s * a.y); }
__device__ __forceinline__ cd cconj(cd a) { return mk(a.x, -a.y); }
__device__ __forceinline__ cd cmul(cd a, cd b) { return mk(fma(a.x, b.x, -(a.y * b.y)), fma(a.x, b.y, a.y * b.x)); }
// a * w for the forward transform (DIR < 0), a * conj(w) for the inverse (DIR > 0); w = forward table entry
template <int DIR> __device__ __forceinline__ cd twmul(cd a, cd w) {
    if (DIR < 0) return mk(fma(a.x, w.x, -(a.y * w.y)), fma(a.x, w.y, a.y * w.x));
    return mk(fma(a.x, w.x, a.y * w.y), fma(a.y, w.x, -(a.x * w.y)));
}
// a * (-i) forward, a * (+i) inverse
template <int DIR> __device__ __forceinline__ cd mul_mi(cd a) {
    if (DIR < 0) return mk(a.y, -a.x);
    return mk(-a.y, a.x);
}

// a * exp(DIR * 2*pi*i * K32/32) for any compile-time K32 in [0, 32): constant 32nd roots of unity
template <int K32, int DIR> __device__ __forceinline__ cd mul_root32(cd a) {
    constexpr double C[16] = {1.0, 0.98078528040323044913, 0.92387953251128675613, 0.83146961230254523708,
                              0.70710678118654752440, 0.55557023301960222474, 0.38268343236508977173,
                              0.19509032201612826785, 0.0, -0.19509032201612826785, -0.38268343236508977173,
                              -0.55557023301960222474, -0.70710678118654752440, -0.83146961230254523708,
                              -0.92387953251128675613, -0.98078528040323044913};
    constexpr double S[16] = {0.0, 0.19509032201612826785, 0.38268343236508977173, 0.55557023301960222474,
                              0.70710678118654752440, 0.83146961230254523708, 0.92387953251128675613,
                              0.98078528040323044913, 1.0, 0.98078528040323044913, 0.92387953251128675613,
                              0.83146961230254523708, 0.70710678118654752440, 0.55557023301960222474,
                              0.38268343236508977173, 0.19509032201612826785};
    constexpr int K = ((K32 % 32) + 32) % 32;
    if constexpr (K >= 16) {
        const cd b = mul_root32<K - 16, DIR>(a);
        return mk(-b.x, -b.y);
    } else if constexpr (K == 0) {
        return a;
    } else if constexpr (K == 8) {
        return (DIR < 0) ? mk(a.y, -a.x) : mk(-a.y, a.x);
    } else {
        constexpr double wr = C[K];
        constexpr double wi = (DIR < 0) ? -S[K] : S[K];
        if constexpr (K == 4) return mk(wr * (a.x + ((DIR < 0) ? a.y : -a.y)), wr * (a.y + ((DIR < 0) ? -a.x : a.x)));
        else return mk(fma(a.x, wr, -(a.y * wi)), fma(a.x, wi, a.y * wr));
    }
}
// a * exp(DIR * 2*pi*i * K/R), R in {2,4,8,16,32}, any integer K >= 0
template <int R, int K, int DIR> __device__ __forceinline__ cd mul_rootN(cd a) {
    static_assert(32 % R == 0, "R must divide 32");
    return mul_root32<(K % R) * (32 / R), DIR>(a);
}

// ---------------------------------------------------------------------------------------------------
// FMA-form radix-2 butterflies.  v = e + W o, vm = e - W o.  The product W o is never formed on its own: its two
// multiply-adds are chained onto e (2 FMA per component), and the mirrored output is vm = 2 e - v (1 FMA per
// component), so a butterfly with a general root costs 6 FMA instead of 4 (product) + 4 (add / subtract).  The
// absolute error of vm is bounded by eps (|e| + |W o|) exactly as for the plain form (it inherits the rounding of
// v), so the backward-error bound of the transform is unchanged.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ cd mirror2(cd e, cd v) { return mk(fma(2.0, e.x, -v.x), fma(2.0, e.y, -v.y)); }

// constant root W = exp(DIR * 2*pi*i * K/R), 0 <= K < R/2, R in {2,4,8,16,32}
template <int R, int K, int DIR> __device__ __forceinline__ void bfly_root(cd e, cd o, cd& v, cd& vm) {
    constexpr int K32 = K * (32 / R);
    constexpr double SQH = 0.70710678118654752440;   // sqrt(1/2)
    // cos / sin (pi m / 16), m = 0..8
    constexpr double CS[9] = {1.0, 0.98078528040323044913, 0.92387953251128675613, 0.83146961230254523708, SQH,
                              0.55557023301960222474, 0.38268343236508977173, 0.19509032201612826785, 0.0};
    if constexpr (K32 == 0) { v = e + o; vm = e - o; }
    else if constexpr (K32 == 8) { const cd t = mul_mi<DIR>(o); v = e + t; vm = e - t; }
    else if constexpr (K32 == 4) {          // W = SQH (1 + sg i):  W o = SQH (o.x - sg o.y, o.y + sg o.x)
        const double dx = (DIR < 0) ? o.x + o.y : o.x - o.y, dy = (DIR < 0) ? o.y - o.x : o.y + o.x;
        v = mk(fma(SQH, dx, e.x), fma(SQH, dy, e.y)); vm = mk(fma(-SQH, dx, e.x), fma(-SQH, dy, e.y));
    } else if constexpr (K32 == 12) {       // W = SQH (-1 + sg i): W o = SQH (-(o.x + sg o.y), sg o.x - o.y)
        const double dx = (DIR < 0) ? o.x - o.y : o.x + o.y, dy = (DIR < 0) ? -o.x - o.y : o.x - o.y;
        v = mk(fma(-SQH, dx, e.x), fma(SQH, dy, e.y)); vm = mk(fma(SQH, dx, e.x), fma(-SQH, dy, e.y));
    } else {                                // angle 2 pi K32 / 32 = pi K32 / 16 in (0, pi)
        constexpr double wr = (K32 < 8) ? CS[K32] : -CS[16 - K32];
        constexpr double wi = ((DIR < 0) ? -1.0 : 1.0) * ((K32 < 8) ? CS[8 - K32] : CS[K32 - 8]);
        v = mk(fma(-o.y, wi, fma(o.x, wr, e.x)), fma(o.y, wr, fma(o.x, wi, e.y)));
        vm = mirror2(e, v);
    }
}

// run-time root: forward (DIR < 0) W = w, inverse W = conj(w), w = forward table entry; ROT: W is additionally
// multiplied by -i (forward) / +i (inverse), i.e. the root a quarter turn further — the same table entry serves both
template <int DIR, bool ROT> __device__ __forceinline__ void bfly_tw(cd e, cd o, cd w, cd& v, cd& vm) {
    if constexpr (DIR < 0 && !ROT) v = mk(fma(-o.y, w.y, fma(o.x, w.x, e.x)), fma(o.y, w.x, fma(o.x, w.y, e.y)));
    else if constexpr (DIR > 0 && !ROT) v = mk(fma(o.y, w.y, fma(o.x, w.x, e.x)), fma(-o.x, w.y, fma(o.y, w.x, e.y)));
    else if constexpr (DIR < 0 && ROT) v = mk(fma(o.y, w.x, fma(o.x, w.y, e.x)), fma(o.y, w.y, fma(-o.x, w.x, e.y)));
    else v = mk(fma(o.x, w.y, fma(-o.y, w.x, e.x)), fma(o.y, w.y, fma(o.x, w.x, e.y)));
    vm = mirror2(e, v);
}

// In-register DFT of R points, natural order in and out:  v[q] <- sum_r v[r] exp(DIR*2*pi*i*r*q/R)
template <int R, int DIR> struct Dft;
template <int DIR> struct Dft<1, DIR> {
    __device__ __forceinline__ static void run(cd*) {}
};
template <int DIR> struct Dft<2, DIR> {
    __device__ __forceinline__ static void run(cd* v) {
        const cd a = v[0], b = v[1];
        v[0] = a + b; v[1] = a - b;
    }
};
template <int DIR> struct Dft<4, DIR> {
    __device__ __forceinline__ static void run(cd* v) {
        const cd a0 = v[0] + v[2], a1 = v[0] - v[2], a2 = v[1] + v[3], a3 = mul_mi<DIR>(v[1] - v[3]);
        v[0] = a0 + a2; v[2] = a0 - a2; v[1] = a1 + a3; v[3] = a1 - a3;
    }
};
template <int R, int K, int DIR> struct Combine {   // v[k] = e[k] + W^k o[k], v[k+R/2] = e[k] - W^k o[k]
    __device__ __forceinline__ static void run(cd* v, const cd* e, const cd* o) {
        bfly_root<R, K, DIR>(e[K], o[K], v[K], v[K + R / 2]);
        if constexpr (K + 1 < R / 2) Combine<R, K + 1, DIR>::run(v, e, o);
    }
};
template <int R, int DIR> struct Dft {
    __device__ __forceinline__ static void run(cd* v) {
        cd e[R / 2], o[R / 2];
#pragma unroll
        for (int i = 0; i < R / 2; ++i) { e[i] = v[2 * i]; o[i] = v[2 * i + 1]; }
        Dft<R / 2, DIR>::run(e);
        Dft<R / 2, DIR>::run(o);
        Combine<R, 0, DIR>::run(v, e, o);
    }
};

// ---------------------------------------------------------------------------------------------------
// Twiddled DFT: v[q] <- sum_r (w^r v[r]) exp(DIR*2*pi*i*r*q/R) with the inter-stage twiddles w^r folded into the
// butterflies.  Decimation in time: y[q] = E[q] + (w W_R^q) O[q], where E, O are the twiddled DFTs of size R/2 of
// the even / odd inputs with base w^2.  Every butterfly then has exactly one run-time root and costs 6 FMA:
// R/2 log2(R) * 6 operations (192 for R = 16) instead of 4 (R-1) for the twiddles plus the plain DFT (60 + 168).
// Roots needed: w W_R^q for q < R/4 (the other quarter is the same entry rotated by -+i), then w^2 W_(R/2)^q, ...:
// R/2 table entries (8 for R = 16) instead of R-1.
// ---------------------------------------------------------------------------------------------------
template <int R> struct TwCount { static constexpr int TOP = (R >= 4) ? R / 4 : 1, value = TOP + TwCount<R / 2>::value; };
template <> struct TwCount<1> { static constexpr int TOP = 0, value = 0; };

// w[] <- the roots of TDft<R>, base exponent m: w = exp(-2*pi*i*m/NT); tw[i*TWS] = exp(-2*pi*i*i/NT)
template <int R, int NT, int TWS> __device__ __forceinline__ void load_tw(cd* w, const cd* __restrict__ tw, int m) {
    if constexpr (R >= 2) {
#pragma unroll
        for (int q = 0; q < TwCount<R>::TOP; ++q) w[q] = __ldg(&tw[(m + q * (NT / R)) * TWS]);
        load_tw<R / 2, NT, TWS>(w + TwCount<R>::TOP, tw, 2 * m);
    }
}
template <int R, int DIR> struct TDft {
    __device__ __forceinline__ static void run(cd* v, const cd* w) {
        if constexpr (R == 2) {
            const cd e = v[0], o = v[1];
            bfly_tw<DIR, false>(e, o, w[0], v[0], v[1]);
        } else {
            cd e[R / 2], o[R / 2];
#pragma unroll
            for (int i = 0; i < R / 2; ++i) { e[i] = v[2 * i]; o[i] = v[2 * i + 1]; }
            TDft<R / 2, DIR>::run(e, w + TwCount<R>::TOP);
            TDft<R / 2, DIR>::run(o, w + TwCount<R>::TOP);
#pragma unroll
            for (int q = 0; q < R / 4; ++q) {
                bfly_tw<DIR, false>(e[q], o[q], w[q], v[q], v[q + R / 2]);
                bfly_tw<DIR, true>(e[q + R / 4], o[q + R / 4], w[q], v[q + R / 4], v[q + R / 4 + R / 2]);
            }
        }
    }
};

// ---------------------------------------------------------------------------------------------------
// line plans: radices per stage and points per thread
// ---------------------------------------------------------------------------------------------------
template <int NL> struct Plan;
template <> struct Plan<4>    { static constexpr int NS = 1, R0 = 4,  R1 = 1,  R2 = 1, E = 4;  };
template <> struct Plan<8>    { static constexpr int NS = 1, R0 = 8,  R1 = 1,  R2 = 1, E = 8;  };
template <> struct Plan<16>   { static constexpr int NS = 2, R0 = 4,  R1 = 4,  R2 = 1, E = 4;  };
template <> struct Plan<32>   { static constexpr int NS = 2, R0 = 8,  R1 = 4,  R2 = 1, E = 8;  };
template <> struct Plan<64>   { static constexpr int NS = 2, R0 = 8,  R1 = 8,  R2 = 1, E = 8;  };
template <> struct Plan<128>  { static constexpr int NS = 2, R0 = 16, R1 = 8,  R2 = 1, E = 16; };
template <> struct Plan<256>  { static constexpr int NS = 2, R0 = 16, R1 = 16, R2 = 1, E = 16; };
template <> struct Plan<512>  { static constexpr int NS = 3, R0 = 8,  R1 = 8,  R2 = 8, E = 16; };
template <> struct Plan<1024> { static constexpr int NS = 3, R0 = 16, R1 = 8,  R2 = 8, E = 16; };

// alternative plan of the 512-point strided passes: ONE shared-memory exchange instead of two (32 points per thread,
// radix 32 then radix 16); chosen per kernel through the PL parameter below
struct Plan512x { static constexpr int NS = 2, R0 = 32, R1 = 16, R2 = 1, E = 32; };

template <int NL, class PL = Plan<NL>> struct PlanInfo {
    typedef PL P;
    static constexpr int E = P::E;
    static constexpr int T = NL / E;    // threads per line
};

// shared-memory tile layouts: element index of (row n, this thread's line)
struct LayoutPlain {        // tile[n][C], thread's column c fixed
    int C, c;
    __device__ __forceinline__ int operator()(int n) const { return n * C + c; }
};
struct LayoutSwz {          // tile[n][SL] with the low 3 slot bits XOR-swizzled by the row (SL >= 8)
    int SL, slot;
    __device__ __forceinline__ int operator()(int n) const { return n * SL + (slot ^ (n & 7)); }
};

// barrier policies of the exchange: the whole CTA, or a named barrier shared by one group of warps (several
// independent transforms per CTA: the TMA-pipelined strided passes)
struct BlockSync {
    __device__ __forceinline__ void operator()() const { __syncthreads(); }
};
struct GroupSync {
    int id, nthreads;       // barrier 1..15, threads of the group (multiple of 32)
    __device__ __forceinline__ void operator()() const { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }
};

// one stage: butterflies on registers; non-final stages scatter to shared memory and gather back
template <int NL, int R, int NSTRIDE /*Ns*/, bool LAST, bool FIRST, int DIR, int TWS, class PL, class Layout, class Sync>
__device__ __forceinline__ void fft_stage(cd (&v)[PL::E], int t, const cd* __restrict__ tw, cd* sm,
                                          const Layout& L, const Sync& sync) {
    constexpr int E = PL::E, T = NL / PL::E, B = E / R;
    static_assert(E % R == 0, "radix must divide the points per thread");
    if constexpr (!LAST && !FIRST) sync();   // every thread has gathered the previous exchange
#pragma unroll
    for (int b = 0; b < B; ++b) {
        const int j = t + b * T;
        const int k = j & (NSTRIDE - 1);
        cd u[R];
#pragma unroll
        for (int r = 0; r < R; ++r) u[r] = v[b + r * B];
        if constexpr (NSTRIDE > 1) {        // inter-stage twiddles w^r, w = exp(-+2 pi i k/(Ns R)), folded into the butterflies
            cd w[TwCount<R>::value];
            load_tw<R, NL, TWS>(w, tw, k * (NL / (NSTRIDE * R)));
            TDft<R, DIR>::run(u, w);
        } else {
            Dft<R, DIR>::run(u);
        }
        if constexpr (LAST) {
#pragma unroll
            for (int q = 0; q < R; ++q) v[b + q * B] = u[q];
        } else {
            const int j0 = (j - k) * R + k;
#pragma unroll
            for (int q = 0; q < R; ++q) sm[L(j0 + q * NSTRIDE)] = u[q];
        }
    }
    if constexpr (!LAST) {
        sync();
#pragma unroll
        for (int m = 0; m < E; ++m) v[m] = sm[L(t + T * m)];
    }
}

// Whole line transform on registers.  On entry v[m] = x[t + T*m]; on exit v[m] = X[t + T*m] with
// X[q] = sum_n x[n] exp(DIR*2*pi*i*n*q/NL) (unnormalised).  `sm` is the exchange tile (must be free on entry;
// all threads of the block — or of the group that `sync` joins — must call).  tw[m*TWS] = exp(-2*pi*i*m/NL).
template <int NL, int DIR, int TWS, class Layout, class Sync = BlockSync, class P = Plan<NL>>
__device__ __forceinline__ void fft_line(cd (&v)[P::E], int t, const cd* __restrict__ tw, cd* sm,
                                         const Layout& L, const Sync& sync = Sync()) {
    if constexpr (P::NS == 1) {
        fft_stage<NL, P::R0, 1, true, true, DIR, TWS, P>(v, t, tw, sm, L, sync);
    } else if constexpr (P::NS == 2) {
        fft_stage<NL, P::R0, 1, false, true, DIR, TWS, P>(v, t, tw, sm, L, sync);
        fft_stage<NL, P::R1, P::R0, true, false, DIR, TWS, P>(v, t, tw, sm, L, sync);
    } else {
        fft_stage<NL, P::R0, 1, false, true, DIR, TWS, P>(v, t, tw, sm, L, sync);
        fft_stage<NL, P::R1, P::R0, false, false, DIR, TWS, P>(v, t, tw, sm, L, sync);
        fft_stage<NL, P::R2, P::R0 * P::R1, true, false, DIR, TWS, P>(v, t, tw, sm, L, sync);
    }
}

}  // namespace mhd

// fft_core.cuh -- register/shared-memory Stockham FFT building blocks for sm_100a.
//
// One transform of length N is owned by T = N/E threads; thread `tid` holds the E elements
// x[tid + T*m], m = 0..E-1, in registers -- before the first pass AND after the last one (the
// Stockham output index of the last pass, jb + t*N/R, is the same ownership pattern), so global
// loads/stores are coalesced and a multi-pass transform needs only (passes-1) shared-memory
// exchanges.  A pass of radix R (R = E, or the remaining factor in the last pass) does E/R
// butterflies per thread:  inputs x[b + t*(E/R)], twiddle w^(t*k) with k = jb mod Ns,
// jb = tid + b*T, outputs to index (jb/Ns)*Ns*R + k + t*Ns.
// WC transforms that are interleaved in memory (a [N][WC] column tile) are handled as one
// transform over vectors: shared index = a*WC + c.
// Exchanges use 64-bit shared accesses; the XOR swizzle below makes every half-warp wavefront
// bank-conflict free for all (N, E, WC) used here (checked by enumeration).
#pragma once
#include <cuda_runtime.h>

namespace tacaw {

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(float2 a, float2 w) {
    return make_float2(fmaf(a.x, w.x, -a.y * w.y), fmaf(a.x, w.y, a.y * w.x));
}
// a * conj(w)
__device__ __forceinline__ float2 cmulc(float2 a, float2 w) {
    return make_float2(fmaf(a.x, w.x, a.y * w.y), fmaf(a.y, w.x, -a.x * w.y));
}
template <bool CONJ>
__device__ __forceinline__ float2 cmul_dir(float2 a, float2 w) {
    return CONJ ? cmulc(a, w) : cmul(a, w);
}
// multiply by -i (forward) or +i (inverse)
template <bool INV>
__device__ __forceinline__ float2 mul_mi(float2 a) {
    return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
}

constexpr __host__ __device__ int ilog2c(int v) { return v <= 1 ? 0 : 1 + ilog2c(v >> 1); }

// ---------------------------------------------------------------------------------------------
// In-register DFTs of size R, natural order in and out.  Forward = exp(-2 pi i st/R).
template <int R, bool INV>
struct Dft;

template <bool INV>
struct Dft<1, INV> {
    static __device__ __forceinline__ void run(float2 (&)[1]) {}
};

template <bool INV>
struct Dft<2, INV> {
    static __device__ __forceinline__ void run(float2 (&v)[2]) {
        float2 a = v[0], b = v[1];
        v[0] = cadd(a, b);
        v[1] = csub(a, b);
    }
};

template <bool INV>
struct Dft<4, INV> {
    static __device__ __forceinline__ void run(float2 (&v)[4]) {
        float2 t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]);
        float2 t2 = cadd(v[1], v[3]), t3 = mul_mi<INV>(csub(v[1], v[3]));
        v[0] = cadd(t0, t2);
        v[1] = cadd(t1, t3);
        v[2] = csub(t0, t2);
        v[3] = csub(t1, t3);
    }
};

template <bool INV>
struct Dft<8, INV> {
    static __device__ __forceinline__ void run(float2 (&v)[8]) {
        float2 e[4] = {v[0], v[2], v[4], v[6]};
        float2 o[4] = {v[1], v[3], v[5], v[7]};
        Dft<4, INV>::run(e);
        Dft<4, INV>::run(o);
        const float c = 0.70710678118654752440f;
        // o1 *= w8, o2 *= w8^2 = -+i, o3 *= w8^3
        float2 o1 = INV ? make_float2(c * (o[1].x - o[1].y), c * (o[1].x + o[1].y))
                        : make_float2(c * (o[1].x + o[1].y), c * (o[1].y - o[1].x));
        float2 o2 = mul_mi<INV>(o[2]);
        float2 o3 = INV ? make_float2(-c * (o[3].x + o[3].y), c * (o[3].x - o[3].y))
                        : make_float2(c * (o[3].y - o[3].x), -c * (o[3].x + o[3].y));
        v[0] = cadd(e[0], o[0]); v[4] = csub(e[0], o[0]);
        v[1] = cadd(e[1], o1);   v[5] = csub(e[1], o1);
        v[2] = cadd(e[2], o2);   v[6] = csub(e[2], o2);
        v[3] = cadd(e[3], o3);   v[7] = csub(e[3], o3);
    }
};

template <bool INV>
struct Dft<16, INV> {
    static __device__ __forceinline__ void run(float2 (&v)[16]) {
        float2 e[8], o[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) { e[i] = v[2 * i]; o[i] = v[2 * i + 1]; }
        Dft<8, INV>::run(e);
        Dft<8, INV>::run(o);
        // w16^k = (cos(k pi/8), -sin(k pi/8)) forward
        const float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f;
        const float c2 = 0.70710678118654752440f;
        const float2 w[8] = {make_float2(1.f, 0.f),  make_float2(c1, -s1),  make_float2(c2, -c2), make_float2(s1, -c1),
                             make_float2(0.f, -1.f), make_float2(-s1, -c1), make_float2(-c2, -c2), make_float2(-c1, -s1)};
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            float2 t = (k == 0) ? o[0] : (k == 4 ? mul_mi<INV>(o[4]) : cmul_dir<INV>(o[k], w[k]));
            v[k] = cadd(e[k], t);
            v[k + 8] = csub(e[k], t);
        }
    }
};

// ---------------------------------------------------------------------------------------------
template <int N, int E>
struct FftPlan {
    static_assert(N >= E && (N & (N - 1)) == 0 && (E == 8 || E == 16), "unsupported FFT plan");
    static constexpr int T = N / E;
    static constexpr __host__ __device__ int radix(int ns) { return (N / ns >= E) ? E : (N / ns); }
    static constexpr __host__ __device__ int ntw_from(int ns) {
        return ns >= N ? 0 : ((ns > 1 ? (radix(ns) - 1) * (E / radix(ns)) : 0) + ntw_from(ns * radix(ns)));
    }
    static constexpr int NTW = ntw_from(1) > 0 ? ntw_from(1) : 1;
    static constexpr int NEXCH = (N > E) ? ((N / E > E) ? 2 + (N / E / E > E ? 1 : 0) : 1) : 0;  // informational
};

// XOR swizzle of a shared index (float2 units); nsw = Ns*WC of the pass that writes.
template <int NSW, int R>
__device__ __forceinline__ int swz(int a) {
    if (NSW >= 16) return a;
    return a ^ (((a >> ilog2c(NSW * R)) << ilog2c(NSW)) & 15);
}

// Fill this thread's twiddle registers from the table roots[j] = exp(-2 pi i j/N) (fp64-accurate).
template <int N, int E, int NS, int OFF>
struct TwInit {
    using P = FftPlan<N, E>;
    static constexpr int R = P::radix(NS);
    static constexpr int NB = E / R;
    static __device__ __forceinline__ void run(float2 (&tw)[P::NTW], const float2* __restrict__ roots, int tid) {
        if constexpr (NS < N) {
            if constexpr (NS > 1) {
#pragma unroll
                for (int b = 0; b < NB; ++b) {
                    int k = (tid + b * P::T) & (NS - 1);
#pragma unroll
                    for (int t = 1; t < R; ++t) tw[OFF + b * (R - 1) + (t - 1)] = roots[t * k * (N / (NS * R))];
                }
            }
            TwInit<N, E, NS * R, OFF + (NS > 1 ? (R - 1) * NB : 0)>::run(tw, roots, tid);
        }
    }
};

// The passes.  x: registers; smA/smB: ping-pong exchange buffers of N*WC float2 each;
// tid in [0,T), c in [0,WC).  TWREG: twiddles from registers `tw`; else from the shared table
// `roots` (N float2).  Sync: functor that synchronises the T*WC threads of this transform group.
template <int N, int E, int WC, bool INV, bool TWREG, int NS, int OFF>
struct FftPass {
    using P = FftPlan<N, E>;
    static constexpr int R = P::radix(NS);
    static constexpr int NB = E / R;
    static constexpr int T = P::T;
    static constexpr bool LAST = (NS * R == N);
    static constexpr int NTWH = (NS > 1) ? (R - 1) * NB : 0;

    template <class Sync>
    static __device__ __forceinline__ void run(float2 (&x)[E], const float2 (&tw)[P::NTW], const float2* roots,
                                               float2* smA, float2* smB, int tid, int c, Sync sync) {
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            float2 v[R];
#pragma unroll
            for (int t = 0; t < R; ++t) v[t] = x[b + t * NB];
            const int jb = tid + b * T;
            const int k = jb & (NS - 1);
            if constexpr (NS > 1) {
#pragma unroll
                for (int t = 1; t < R; ++t) {
                    float2 w;
                    if constexpr (TWREG) w = tw[OFF + b * (R - 1) + (t - 1)];
                    else w = roots[t * k * (N / (NS * R))];
                    v[t] = cmul_dir<INV>(v[t], w);
                }
            }
            Dft<R, INV>::run(v);
            if constexpr (LAST) {
#pragma unroll
                for (int t = 0; t < R; ++t) x[b + t * NB] = v[t];
            } else {
                const int base = (jb - k) * R + k;
#pragma unroll
                for (int t = 0; t < R; ++t) smA[swz<NS * WC, R>((base + t * NS) * WC + c)] = v[t];
            }
        }
        if constexpr (!LAST) {
            sync();
#pragma unroll
            for (int m = 0; m < E; ++m) x[m] = smA[swz<NS * WC, R>((tid + T * m) * WC + c)];
            FftPass<N, E, WC, INV, TWREG, NS * R, OFF + NTWH>::run(x, tw, roots, smB, smA, tid, c, sync);
        }
    }
};

template <int N, int E, int WC, bool INV, bool TWREG, class Sync>
__device__ __forceinline__ void fft_regs(float2 (&x)[E], const float2 (&tw)[FftPlan<N, E>::NTW], const float2* roots,
                                         float2* smA, float2* smB, int tid, int c, Sync sync) {
    FftPass<N, E, WC, INV, TWREG, 1, 0>::run(x, tw, roots, smA, smB, tid, c, sync);
}

// number of exchanges of a plan (so callers know which ping-pong buffer the next transform may use)
template <int N, int E>
constexpr int fft_nexch() {
    int n = 0;
    for (int ns = 1; ns < N;) {
        int r = FftPlan<N, E>::radix(ns);
        if (ns * r < N) ++n;
        ns *= r;
    }
    return n;
}

struct SyncWarp {
    __device__ __forceinline__ void operator()() const { __syncwarp(); }
};
struct SyncBlock {
    __device__ __forceinline__ void operator()() const { __syncthreads(); }
};
struct SyncNamed {
    int id, count;
    __device__ __forceinline__ void operator()() const { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }
};

}  // namespace tacaw

// fft2.cuh -- single-exchange register FFTs for the multislice slice step (sm_100a).
//
// The slice-step kernels are bound by the L1TEX unit (shared-memory wavefronts + global tag stage, ncu
// profiles/r1_*), not by HBM or the FMA pipe, so a transform here moves every element through shared
// memory as few times as possible: thread `tid` of the T = N/E threads that own a transform holds the
// E = 32 (N >= 512), 16 (N >= 128) or 8 elements x[tid + T*m]; the first pass is one radix-E DFT in
// registers, ONE padded shared-memory exchange follows, and the second pass does E/R radix-R DFTs
// (R = N/E) with twiddles read from a per-thread-slot table in shared memory (a warp that holds two
// rows reads each twiddle as a broadcast).  N = 2048 = 32*32*2 needs a second exchange.  Ownership is
// x[tid + T*m] before the first pass and after the last one, so global accesses are coalesced.
// Complex multiplies are two packed fp32x2 instructions (cmul / cmulc in fft_core.cuh).
#pragma once
#include <cmath>
#include <type_traits>

#include "fft_core.cuh"

namespace tacaw {

// ---------------------------------------------------------------------------------------------
// 32-point DFT in registers: two 16-point DFTs and one combine stage with W32^k.
template <bool INV, bool SOUT>
struct Dft<32, INV, SOUT> {
    static __device__ __forceinline__ void run(float2 (&v)[32]) {
        float2 e[16], o[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) { e[i] = v[2 * i]; o[i] = v[2 * i + 1]; }
        Dft<16, INV, false>::run(e);
        Dft<16, INV, false>::run(o);
        // cos(pi k/16), k = 0..8
        constexpr float C[9] = {1.0f, 0.98078528040323044913f, 0.92387953251128675613f, 0.83146961230254523708f,
                                0.70710678118654752440f, 0.55557023301960222474f, 0.38268343236508977173f,
                                0.19509032201612826785f, 0.0f};
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            if (k == 0) {
                v[0] = cadd(e[0], o[0]);  v[16] = csub(e[0], o[0]);
            } else if (k == 8) {
                v[8] = add_mi<INV>(e[8], o[8]);  v[24] = sub_mi<INV>(e[8], o[8]);
            } else if (k == 4) {      // W = c(1 -+ i)
                float2 t = add_mi<INV>(o[4], o[4]);
                v[4] = axpy(C[4], t, e[4]);  v[20] = axpy(-C[4], t, e[4]);
            } else if (k == 12) {     // W = -c(1 +- i)
                float2 t = sub_mi<INV>(o[12], o[12]);
                v[12] = axpy(-C[4], t, e[12]);  v[28] = axpy(C[4], t, e[12]);
            } else {
                // forward W32^k = (cos(pi k/16), -sin(pi k/16))
                const float wr = (k < 8) ? C[k] : -C[16 - k];
                const float wi = (k < 8) ? C[8 - k] : C[k - 8];
                float2 t = cmul_dir<INV>(o[k], make_float2(wr, -wi));
                v[k] = cadd(e[k], t);  v[k + 16] = csub(e[k], t);
            }
        }
    }
};

// ---------------------------------------------------------------------------------------------
// Plan: elements per thread and pass structure.
constexpr __host__ __device__ int fft2_elems(int n) { return n >= 512 ? 32 : (n >= 128 ? 16 : 8); }

template <int N>
struct Plan2 {
    static constexpr int E = fft2_elems(N);
    static constexpr int T = N / E;
    static_assert(N >= 16 && (N & (N - 1)) == 0 && T >= 1, "unsupported size");
    static constexpr __host__ __device__ int radix(int ns) { return (N / ns >= E) ? E : (N / ns); }
    // twiddle slots of the passes from `ns` on: (R-1) per butterfly, E/R butterflies per thread
    static constexpr __host__ __device__ int slots_from(int ns) {
        return ns >= N ? 0 : ((ns > 1 ? (radix(ns) - 1) * (E / radix(ns)) : 0) + slots_from(ns * radix(ns)));
    }
    static constexpr int NSLOT = slots_from(1);
    static constexpr int TW_ELEMS = NSLOT * T;     // float2 entries of the shared twiddle table
};

// Exchange buffer: the pass with Ns = 1 writes E consecutive vector elements per thread; one pad of WC
// elements per thread makes the half-warp wavefronts of those writes and of the (contiguous) reads
// bank-conflict free.  Later exchanges (N = 2048 only) are conflict free unpadded.
constexpr __host__ __device__ int exch2_elems(int n, int wc) { return n * wc + (n / fft2_elems(n)) * wc; }

// Twiddle table, entry (slot, tid) = root^(t k N/(Ns R)), k = (tid + b T) mod Ns, for the passes with
// Ns > 1 in order, butterflies b, inputs t = 1..R-1; root = exp(-2 pi i/N).  Built once per context on the
// host in fp64 (fft2_host_table), copied to shared memory by every CTA (fft2_load_twiddles).
inline int fft2_table_elems(int n) {
    const int e = fft2_elems(n), t = n / e;
    int slots = 0;
    for (int ns = e; ns < n;) {
        const int r = (n / ns >= e) ? e : n / ns;
        slots += (r - 1) * (e / r);
        ns *= r;
    }
    return slots * t;
}
template <class F2>
inline void fft2_host_table(int n, F2* tab) {
    const int e = fft2_elems(n), T = n / e;
    int slot0 = 0;
    for (int ns = e; ns < n;) {
        const int r = (n / ns >= e) ? e : n / ns;
        for (int b = 0; b < e / r; ++b)
            for (int t = 1; t < r; ++t)
                for (int tid = 0; tid < T; ++tid) {
                    const int k = (tid + b * T) & (ns - 1);
                    const long long idx = ((long long)t * k * (n / (ns * r))) % n;
                    const double ang = -2.0 * 3.14159265358979323846 * (double)idx / (double)n;
                    F2 v;
                    v.x = (float)cos(ang);
                    v.y = (float)sin(ang);
                    tab[(size_t)(slot0 + b * (r - 1) + (t - 1)) * T + tid] = v;
                }
        slot0 += (r - 1) * (e / r);
        ns *= r;
    }
}
template <int N>
__device__ __forceinline__ void fft2_load_twiddles(float2* __restrict__ tab, const float2* __restrict__ gtab, int lt,
                                                   int nthreads) {
    static_assert(Plan2<N>::TW_ELEMS % 2 == 0, "table is copied in 16-byte chunks");
    for (int i = lt; i < Plan2<N>::TW_ELEMS / 2; i += nthreads) cp_async16(tab + 2 * i, gtab + 2 * i);
    cp_async_commit();
}

// ---------------------------------------------------------------------------------------------
// The passes.  x: registers.  twp = table + tid.  ex: exchange buffer of exch2_elems(N, WC) float2.
// (tid, c): transform thread and interleaved-column index.  Sync synchronises the threads that share the
// buffer.  PRESYNC: also synchronise before writing (the buffer may still be read by a previous exchange).
template <int N, int WC, bool INV, bool PRESYNC, int NS, int SLOT>
struct Pass2 {
    using P = Plan2<N>;
    static constexpr int E = P::E, T = P::T;
    static constexpr int R = P::radix(NS);
    static constexpr int NB = E / R;
    static constexpr bool LAST = (NS * R == N);
    static constexpr int NSL = (NS > 1) ? (R - 1) * NB : 0;
    static constexpr bool PAD = (NS == 1);
    static_assert(LAST || PAD || NS * WC >= 16, "unpadded exchange would conflict");
    // pad: +WC elements per block of E*WC (the block one thread writes in the first pass)
    static constexpr __host__ __device__ int rpad(int m) {     // read offset of element m (tid part excluded)
        return T * m * WC + (PAD ? ((T >= E) ? (T / E) * m : m / (E / T)) * WC : 0);
    }

    // hook(): called once, right after the registers were refilled from the LAST exchange of the transform
    // (the buffer is then free as soon as the sharing threads have synchronised)
    template <class Sync, class Hook>
    static __device__ __forceinline__ void run(float2 (&x)[E], const float2* __restrict__ twp, float2* ex, int tid, int c,
                                               Sync& sync, Hook& hook) {
        if constexpr (!LAST && PRESYNC) sync();
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            float2 v[R];
#pragma unroll
            for (int t = 0; t < R; ++t) v[t] = x[b + t * NB];
            if constexpr (NS > 1) {
#pragma unroll
                for (int t = 1; t < R; ++t) v[t] = cmul_dir<INV>(v[t], twp[(SLOT + b * (R - 1) + (t - 1)) * T]);
            }
            Dft<R, INV, false>::run(v);
            if constexpr (LAST) {
#pragma unroll
                for (int t = 0; t < R; ++t) x[b + t * NB] = v[t];
            } else {
                const int jb = tid + b * T, k = jb & (NS - 1);
                float2* wp = ex + ((jb - k) * R + k) * WC + c + (PAD ? jb * WC : 0);
#pragma unroll
                for (int t = 0; t < R; ++t) wp[t * NS * WC] = v[t];
            }
        }
        if constexpr (!LAST) {
            if constexpr (NS == 1) hook.pre();
            sync();
            const float2* rp = ex + tid * WC + c + (PAD && T >= E ? (tid / E) * WC : 0);
#pragma unroll
            for (int m = 0; m < E; ++m) x[m] = rp[rpad(m)];
            using Next = Pass2<N, WC, INV, true, NS * R, SLOT + NSL>;
            if constexpr (Next::LAST) hook();
            Next::run(x, twp, ex, tid, c, sync, hook);
        }
    }
};

// Hooks of a transform: pre() runs right before the barrier of the first exchange (after this thread's
// writes), operator() right after the registers were refilled from the last exchange.
struct NoHook {
    __device__ __forceinline__ void pre() const {}
    __device__ __forceinline__ void operator()() const {}
};
template <class Pre, class Post>
struct Hooks {
    Pre pre_;
    Post post_;
    __device__ __forceinline__ void pre() { pre_(); }
    __device__ __forceinline__ void operator()() { post_(); }
};

// One transform of length N over WC interleaved columns; PRESYNC as above for the first exchange.
template <int N, int WC, bool INV, bool PRESYNC, class Sync, class Hook>
__device__ __forceinline__ void fft2(float2 (&x)[Plan2<N>::E], const float2* __restrict__ twp, float2* ex, int tid, int c,
                                     Sync& sync, Hook& hook) {
    Pass2<N, WC, INV, PRESYNC, 1, 0>::run(x, twp, ex, tid, c, sync, hook);
}
template <int N, int WC, bool INV, bool PRESYNC, class Sync>
__device__ __forceinline__ void fft2(float2 (&x)[Plan2<N>::E], const float2* __restrict__ twp, float2* ex, int tid, int c,
                                     Sync& sync) {
    NoHook h;
    Pass2<N, WC, INV, PRESYNC, 1, 0>::run(x, twp, ex, tid, c, sync, h);
}

// ---------------------------------------------------------------------------------------------
// N = 2048 with ONE shared-memory exchange per transform (the "pair plan").  The T = 64 threads that own a transform are 32
// lane pairs, tq = tid >> 1, odd = tid & 1.  Even lanes run the 1024-point transform of the even samples, odd lanes that
// of the odd samples -- with ownership x[tid + 64 m] these are exactly the two interleaved columns of ONE
// fft2<1024, 2 WC> call (column = lane parity) -- and a radix-2 stage ACROSS the lane pair replaces the third pass and
// its exchange: 16 values per thread change hands through SHFL.xor, the other 16 stay.
//   fft2x_dit (decimation in time, first transform of a kernel):
//       canonical ownership x[tid + 64 m] in;  S0, S1 = transforms of the even / odd samples;
//       X[k] = S0[k] + w^k S1[k],  X[k + 1024] = S0[k] - w^k S1[k],  w = exp(-+2 pi i/2048)
//       PAIRED ownership out:  x[m] = X[kq + 32 m],  x[16 + m] = X[kq + 32 m + 1024],  m < 16,  kq = tq + 512 odd
//   fft2x_dif (decimation in frequency, second transform of a kernel):
//       paired ownership in;  a[n] = x[n] + x[n + 1024],  b[n] = (x[n] - x[n + 1024]) w^n;
//       even lanes transform a (X[2k]), odd lanes b (X[2k + 1]);  canonical ownership out.
// So a kernel that does two transforms with a pointwise product between them loads and stores coalesced rows exactly as
// the single-exchange plans do, and the product is taken in the paired ownership.
// cwp = combine table + tid, entry (m, tid) = exp(-2 pi i (kq + 32 m)/2048), 16 x 64 entries (pair_host_table).
constexpr int PAIR_N = 2048;
constexpr int PAIR_T = 64;                      // threads per transform
constexpr int PAIR_CW_ELEMS = 16 * PAIR_T;      // combine-twiddle table entries

// index of register m in the paired ownership (kq = tq + 512 odd)
constexpr __host__ __device__ int pair_off(int m) { return 32 * (m & 15) + ((m >= 16) ? 1024 : 0); }

template <class F2>
inline void pair_host_table(F2* tab) {
    for (int m = 0; m < 16; ++m)
        for (int tid = 0; tid < PAIR_T; ++tid) {
            const int k = (tid >> 1) + 512 * (tid & 1) + 32 * m;
            const double ang = -2.0 * 3.14159265358979323846 * (double)k / (double)PAIR_N;
            F2 v;
            v.x = (float)cos(ang);
            v.y = (float)sin(ang);
            tab[m * PAIR_T + tid] = v;
        }
}

__device__ __forceinline__ float2 shfl_xor2(float2 v, int mask) {
    return make_float2(__shfl_xor_sync(0xffffffffu, v.x, mask), __shfl_xor_sync(0xffffffffu, v.y, mask));
}
__device__ __forceinline__ float2 sel2(bool c, float2 a, float2 b) { return make_float2(c ? a.x : b.x, c ? a.y : b.y); }

// Combine twiddle w^(kq + 32 m) of register pair m: from the 16 x 64 table (shared memory or global/L1) ...
struct PairTwTable {
    const float2* cwp;      // table + tid
    __device__ __forceinline__ float2 operator()(int m) const { return cwp[m * PAIR_T]; }
};
// ... or computed: w^kq (two registers, read once per kernel) times the compile-time constant w^(32 m) = exp(-2 pi i m/64).
// Costs one more complex multiply per pair but no memory access.
struct PairTwCompute {
    float2 wb;              // w^kq
    __device__ __forceinline__ float2 operator()(int m) const {
        constexpr float C64[17] = {1.0f, 0.99518472667219688624f, 0.98078528040323044913f, 0.95694033573220886494f,
                                   0.92387953251128675613f, 0.88192126434835502971f, 0.83146961230254523708f,
                                   0.77301045336273696081f, 0.70710678118654752440f, 0.63439328416364549822f,
                                   0.55557023301960222474f, 0.47139673682599764856f, 0.38268343236508977173f,
                                   0.29028467725446236764f, 0.19509032201612826785f, 0.09801714032956060199f, 0.0f};
        if (m == 0) return wb;
        return cmul(wb, make_float2(C64[m], -C64[16 - m]));     // exp(-2 pi i m/64) = (cos, -sin), sin(2 pi m/64) = cos(2 pi (16-m)/64)
    }
};

// twq = 1024-point twiddle table + tq;  ex: exchange buffer of exch2_elems(1024, 2 WC);  cc = column index of this thread
// among the 2 WC interleaved sub-transforms (= lt & (2 WC - 1) with lt = tid WC + c);  the lane partner is lane ^ WC.
template <int WC, bool INV, bool PRESYNC, class CW, class Sync, class Hook>
__device__ __forceinline__ void fft2x_dit(float2 (&x)[32], const float2* __restrict__ twq, const CW& cw,
                                          float2* ex, int tq, int cc, bool odd, Sync& sync, Hook& hook) {
    fft2<1024, 2 * WC, INV, PRESYNC>(x, twq, ex, tq, cc, sync, hook);
#pragma unroll
    for (int m = 0; m < 16; ++m) {
        // the even lane finishes k = tq + 32 m, the odd lane k = tq + 32 (m + 16): each sends what the other needs
        const float2 recv = shfl_xor2(sel2(odd, x[m], x[m + 16]), WC);
        const float2 a = sel2(odd, recv, x[m]);              // S0[k]
        const float2 b = sel2(odd, x[m + 16], recv);         // S1[k]
        const float2 bt = cmul_dir<INV>(b, cw(m));
        x[m] = cadd(a, bt);
        x[m + 16] = csub(a, bt);
    }
}

template <int WC, bool INV, bool PRESYNC, class CW, class Sync, class Hook>
__device__ __forceinline__ void fft2x_dif(float2 (&x)[32], const float2* __restrict__ twq, const CW& cw,
                                          float2* ex, int tq, int cc, bool odd, Sync& sync, Hook& hook) {
#pragma unroll
    for (int m = 0; m < 16; ++m) {
        const float2 u = cadd(x[m], x[m + 16]);                                   // a[kq + 32 m]
        const float2 v = cmul_dir<INV>(csub(x[m], x[m + 16]), cw(m));              // b[kq + 32 m]
        // even lanes collect a[tq + 32 m'], odd lanes b[tq + 32 m'], m' = 0..31
        const float2 recv = shfl_xor2(sel2(odd, u, v), WC);
        x[m] = sel2(odd, recv, u);
        x[m + 16] = sel2(odd, v, recv);
    }
    fft2<1024, 2 * WC, INV, PRESYNC>(x, twq, ex, tq, cc, sync, hook);
}

// Plan of the slice-step kernels for a transform length N: the single-exchange plan, or the pair plan at 2048.
template <int N>
struct XPlan {
    static constexpr bool PAIR = (N == PAIR_N);
    static constexpr int NSUB = PAIR ? N / 2 : N;                 // length of the shared-memory transforms
    using P = Plan2<NSUB>;
    static constexpr int E = P::E;
    static constexpr int T = N / E;                               // threads per transform
    static constexpr int TW_ELEMS = P::TW_ELEMS + (PAIR ? PAIR_CW_ELEMS : 0);
    static constexpr __host__ __device__ int exch(int wc) { return PAIR ? exch2_elems(NSUB, 2 * wc) : exch2_elems(N, wc); }
};
inline int xplan_table_elems(int n) { return n == PAIR_N ? fft2_table_elems(n / 2) + PAIR_CW_ELEMS : fft2_table_elems(n); }
template <class F2>
inline void xplan_host_table(int n, F2* tab) {
    if (n == PAIR_N) {
        fft2_host_table(n / 2, tab);
        pair_host_table(tab + fft2_table_elems(n / 2));
    } else {
        fft2_host_table(n, tab);
    }
}
// CW_SMEM = false: only the sub-transform twiddles go to shared memory, the combine table stays in global memory (L1)
template <int N, bool CW_SMEM = true>
__device__ __forceinline__ void xplan_load_twiddles(float2* __restrict__ tab, const float2* __restrict__ gtab, int lt, int nthreads) {
    constexpr int NE = CW_SMEM ? XPlan<N>::TW_ELEMS : XPlan<N>::P::TW_ELEMS;
    static_assert(NE % 2 == 0, "table is copied in 16-byte chunks");
    for (int i = lt; i < NE / 2; i += nthreads) cp_async16(tab + 2 * i, gtab + 2 * i);
    cp_async_commit();
}

// Per-thread view of a plan: transform thread index, twiddle pointers, and the index of register m in the ownership
// BETWEEN the two transforms of a kernel (canonical tid + T m, or the paired ownership at 2048).
template <int N, int WC, bool CW_COMPUTE = false>
struct XThread {
    using X = XPlan<N>;
    using CWT = typename std::conditional<CW_COMPUTE, PairTwCompute, PairTwTable>::type;
    const float2* twp;      // sub-transform twiddles of this thread
    CWT cwt;                // combine twiddles (pair plan)
    int tid, c;             // transform thread, column of the tile
    int tq, cc;             // pair plan: sub-transform thread and interleaved column
    bool odd;
    int mid0;               // index of register 0 between the transforms
    // tw: twiddle table in shared memory; cw: the combine table of the pair plan (shared or global memory)
    __device__ __forceinline__ XThread(const float2* tw, const float2* cw, int tid_, int c_) : tid(tid_), c(c_) {
        if constexpr (X::PAIR) {
            tq = tid >> 1;
            odd = (tid & 1) != 0;
            cc = (tid & 1) * WC + c;
            twp = tw + tq;
            if constexpr (CW_COMPUTE) cwt.wb = cw[tid];          // row m = 0 of the table: w^kq
            else cwt.cwp = cw + tid;
            mid0 = tq + (odd ? 512 : 0);
        } else {
            tq = tid; cc = c; odd = false;
            twp = tw + tid;
            mid0 = tid;
        }
    }
    static constexpr __host__ __device__ int mid_off(int m) { return X::PAIR ? pair_off(m) : X::T * m; }
    __device__ __forceinline__ int mid(int m) const { return mid0 + mid_off(m); }
    // first transform of a kernel: canonical ownership in, `mid` ownership out
    template <bool INV, bool PRESYNC, class Sync, class Hook>
    __device__ __forceinline__ void first(float2 (&x)[X::E], float2* ex, Sync& sync, Hook& hook) const {
        if constexpr (X::PAIR) fft2x_dit<WC, INV, PRESYNC>(x, twp, cwt, ex, tq, cc, odd, sync, hook);
        else fft2<N, WC, INV, PRESYNC>(x, twp, ex, tid, c, sync, hook);
    }
    // second transform of a kernel: `mid` ownership in, canonical ownership out
    template <bool INV, bool PRESYNC, class Sync, class Hook>
    __device__ __forceinline__ void second(float2 (&x)[X::E], float2* ex, Sync& sync, Hook& hook) const {
        if constexpr (X::PAIR) fft2x_dif<WC, INV, PRESYNC>(x, twp, cwt, ex, tq, cc, odd, sync, hook);
        else fft2<N, WC, INV, PRESYNC>(x, twp, ex, tid, c, sync, hook);
    }
};

}  // namespace tacaw

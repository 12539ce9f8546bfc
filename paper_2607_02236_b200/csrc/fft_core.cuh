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
// Exchanges use 64-bit shared accesses into a padded buffer, index P(A) = A + ((A >> 4) << u): the
// pad makes every half-warp wavefront bank-conflict free for all (N, E, WC) used here AND keeps the
// per-output / per-element offsets additive compile-time constants (both checked by enumeration,
// see DESIGN.md), so an exchange costs one base address computation plus immediate offsets.
// Butterflies use the sm_100 packed fp32x2 instructions (FADD2 / FFMA2): a complex add is one
// instruction and the +-i rotations ride on FADD2's operand swizzle (LO_HI.NP) for free.
#pragma once
#include <cuda_runtime.h>

namespace tacaw {

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
// complex multiply as two packed instructions: FMUL2 with a broadcast scalar operand, then FFMA2 whose
// first operand is the swapped / half-negated register pair (an operand modifier, no extra MOV)
__device__ __forceinline__ float2 cmul(float2 a, float2 w) {
    float2 r = __fmul2_rn(a, make_float2(w.x, w.x));
    return __ffma2_rn(make_float2(-a.y, a.x), make_float2(w.y, w.y), r);
}
// a * conj(w)
__device__ __forceinline__ float2 cmulc(float2 a, float2 w) {
    float2 r = __fmul2_rn(a, make_float2(w.x, w.x));
    return __ffma2_rn(make_float2(a.y, -a.x), make_float2(w.y, w.y), r);
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
// scalar variants for values that are stored right away: ptxas puts a MOV pair between a packed
// FADD2/FFMA2 result and an STS/STG that consumes it, so the last butterfly stage before a store
// is cheaper in scalar fp32 (2 FADD) than packed (FADD2 + 2 MOV)
template <bool S>
__device__ __forceinline__ float2 caddS(float2 a, float2 b) {
    return S ? make_float2(a.x + b.x, a.y + b.y) : __fadd2_rn(a, b);
}
template <bool S>
__device__ __forceinline__ float2 csubS(float2 a, float2 b) {
    return S ? make_float2(a.x - b.x, a.y - b.y) : __fadd2_rn(a, make_float2(-b.x, -b.y));
}
template <bool S>
__device__ __forceinline__ float2 axpyS(float s, float2 t, float2 e) {
    return S ? make_float2(fmaf(s, t.x, e.x), fmaf(s, t.y, e.y)) : __ffma2_rn(t, make_float2(s, s), e);
}
// a + (-+i) b  and  a - (-+i) b  (one FADD2 each: the rotation is an operand swizzle)
template <bool INV, bool S = false>
__device__ __forceinline__ float2 add_mi(float2 a, float2 b) { return caddS<S>(a, mul_mi<INV>(b)); }
template <bool INV, bool S = false>
__device__ __forceinline__ float2 sub_mi(float2 a, float2 b) { return caddS<S>(a, mul_mi<!INV>(b)); }
// e + s*t (s real)
__device__ __forceinline__ float2 axpy(float s, float2 t, float2 e) { return __ffma2_rn(t, make_float2(s, s), e); }

constexpr __host__ __device__ int ilog2c(int v) { return v <= 1 ? 0 : 1 + ilog2c(v >> 1); }

// ---------------------------------------------------------------------------------------------
// In-register DFTs of size R, natural order in and out.  Forward = exp(-2 pi i st/R).
// SOUT: the outputs are stored right away (scalar last stage, see caddS).
template <int R, bool INV, bool SOUT = false>
struct Dft;

template <bool INV, bool SOUT>
struct Dft<1, INV, SOUT> {
    static __device__ __forceinline__ void run(float2 (&)[1]) {}
};

template <bool INV, bool SOUT>
struct Dft<2, INV, SOUT> {
    static __device__ __forceinline__ void run(float2 (&v)[2]) {
        float2 a = v[0], b = v[1];
        v[0] = caddS<SOUT>(a, b);
        v[1] = csubS<SOUT>(a, b);
    }
};

template <bool INV, bool SOUT>
struct Dft<4, INV, SOUT> {
    static __device__ __forceinline__ void run(float2 (&v)[4]) {
        float2 t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]);
        float2 t2 = cadd(v[1], v[3]), t3 = csub(v[1], v[3]);
        v[0] = caddS<SOUT>(t0, t2);
        v[2] = csubS<SOUT>(t0, t2);
        v[1] = add_mi<INV, SOUT>(t1, t3);
        v[3] = sub_mi<INV, SOUT>(t1, t3);
    }
};

template <bool INV, bool SOUT>
struct Dft<8, INV, SOUT> {
    static __device__ __forceinline__ void run(float2 (&v)[8]) {
        float2 e[4] = {v[0], v[2], v[4], v[6]};
        float2 o[4] = {v[1], v[3], v[5], v[7]};
        Dft<4, INV, false>::run(e);
        Dft<4, INV, false>::run(o);
        const float c = 0.70710678118654752440f;
        // o1 w8 = c (o1 + (-+i) o1);   o3 w8^3 = -c (o3 - (-+i) o3)
        float2 t1 = add_mi<INV>(o[1], o[1]);
        float2 t3 = sub_mi<INV>(o[3], o[3]);
        v[0] = caddS<SOUT>(e[0], o[0]);        v[4] = csubS<SOUT>(e[0], o[0]);
        v[1] = axpyS<SOUT>(c, t1, e[1]);       v[5] = axpyS<SOUT>(-c, t1, e[1]);
        v[2] = add_mi<INV, SOUT>(e[2], o[2]);  v[6] = sub_mi<INV, SOUT>(e[2], o[2]);
        v[3] = axpyS<SOUT>(-c, t3, e[3]);      v[7] = axpyS<SOUT>(c, t3, e[3]);
    }
};

template <bool INV, bool SOUT>
struct Dft<16, INV, SOUT> {
    static __device__ __forceinline__ void run(float2 (&v)[16]) {
        float2 e[8], o[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) { e[i] = v[2 * i]; o[i] = v[2 * i + 1]; }
        Dft<8, INV, false>::run(e);
        Dft<8, INV, false>::run(o);
        // w16^k = (cos(k pi/8), -sin(k pi/8)) forward
        const float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f;
        const float c2 = 0.70710678118654752440f;
        constexpr bool S = SOUT;
        v[0] = caddS<S>(e[0], o[0]);  v[8] = csubS<S>(e[0], o[0]);
        {   float2 t = cmul_dir<INV>(o[1], make_float2(c1, -s1));  v[1] = caddS<S>(e[1], t);  v[9] = csubS<S>(e[1], t); }
        {   float2 t = add_mi<INV>(o[2], o[2]);  v[2] = axpyS<S>(c2, t, e[2]);  v[10] = axpyS<S>(-c2, t, e[2]); }
        {   float2 t = cmul_dir<INV>(o[3], make_float2(s1, -c1));  v[3] = caddS<S>(e[3], t);  v[11] = csubS<S>(e[3], t); }
        v[4] = add_mi<INV, S>(e[4], o[4]);  v[12] = sub_mi<INV, S>(e[4], o[4]);
        {   float2 t = cmul_dir<INV>(o[5], make_float2(-s1, -c1)); v[5] = caddS<S>(e[5], t);  v[13] = csubS<S>(e[5], t); }
        {   float2 t = sub_mi<INV>(o[6], o[6]);  v[6] = axpyS<S>(-c2, t, e[6]);  v[14] = axpyS<S>(c2, t, e[6]); }
        {   float2 t = cmul_dir<INV>(o[7], make_float2(-c1, -s1)); v[7] = caddS<S>(e[7], t);  v[15] = csubS<S>(e[7], t); }
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

// Padded shared index P(A) = A + ((A >> 4) << u) for the exchange written by the pass (NS, R) of
// a transform over WC interleaved columns; u < 0 means no pad.  Rule found by exhaustive search:
// conflict-free writes and reads per half-warp, offsets additive (see header comment).
constexpr __host__ __device__ int pad_u(int wc, int ns, int r) {
    return (ns * wc >= 16) ? -1 : (wc == 1 ? (ns == 1 ? 0 : 1) : (r == 8 ? 1 : 0));
}
constexpr __host__ __device__ int pad_idx(int a, int u) { return u < 0 ? a : a + ((a >> 4) << u); }
// float2 elements an exchange buffer needs for a transform of n points over wc columns
constexpr __host__ __device__ int exch_elems(int n, int wc) { return n * wc + (n * wc) / 8; }

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
template <int N, int E, int WC, bool INV, bool TWREG, bool STORE_AFTER, int NS, int OFF>
struct FftPass {
    using P = FftPlan<N, E>;
    static constexpr int R = P::radix(NS);
    static constexpr int NB = E / R;
    static constexpr int T = P::T;
    static constexpr bool LAST = (NS * R == N);
    static constexpr int NTWH = (NS > 1) ? (R - 1) * NB : 0;

    static constexpr int U = pad_u(WC, NS, R);
    // compile-time offsets relative to the padded base (thread-independent by construction)
    static constexpr __host__ __device__ int woff(int b, int t) {
        const int b0 = b * T, k0 = b0 & (NS - 1), base0 = ((b0 - k0) * R + k0) * WC;
        return pad_idx(base0 + t * NS * WC, U) - pad_idx(base0, U);
    }
    static constexpr __host__ __device__ int roff(int m) { return pad_idx(T * m * WC, U); }

    template <class Sync>
    static __device__ __forceinline__ void run(float2 (&x)[E], const float2 (&tw)[P::NTW], const float2* roots,
                                               float2* smA, float2* smB, int tid, int c, Sync& sync) {
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
            Dft<R, INV, (!LAST) || STORE_AFTER>::run(v);
            if constexpr (LAST) {
#pragma unroll
                for (int t = 0; t < R; ++t) x[b + t * NB] = v[t];
            } else {
                float2* wp = smA + pad_idx(((jb - k) * R + k) * WC + c, U);
#pragma unroll
                for (int t = 0; t < R; ++t) wp[woff(b, t)] = v[t];
            }
        }
        if constexpr (!LAST) {
            sync();
            const float2* rp = smA + pad_idx(tid * WC + c, U);
#pragma unroll
            for (int m = 0; m < E; ++m) x[m] = rp[roff(m)];
            FftPass<N, E, WC, INV, TWREG, STORE_AFTER, NS * R, OFF + NTWH>::run(x, tw, roots, smB, smA, tid, c, sync);
        }
    }
};

// STORE_AFTER: the transform's outputs go straight to a global store (no arithmetic in between).
template <int N, int E, int WC, bool INV, bool TWREG, bool STORE_AFTER = false, class Sync>
__device__ __forceinline__ void fft_regs(float2 (&x)[E], const float2 (&tw)[FftPlan<N, E>::NTW], const float2* roots,
                                         float2* smA, float2* smB, int tid, int c, Sync& sync) {
    FftPass<N, E, WC, INV, TWREG, STORE_AFTER, 1, 0>::run(x, tw, roots, smA, smB, tid, c, sync);
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

// 16-byte asynchronous global -> shared copy (LDGSTS), bypassing L1 and registers.
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
// the same with an L2 eviction-priority hint (createpolicy): streamed-once data (the t_n rows) is marked evict_first so
// that it does not displace the waves of the L2-resident groups
__device__ __forceinline__ unsigned long long l2_policy_evict_first() {
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ unsigned long long l2_policy_evict_last() {
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void cp_async16_hint(void* smem_dst, const void* gmem_src, unsigned long long policy) {
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"(d), "l"(gmem_src), "l"(policy) : "memory");
}
// 8-byte variant (one complex64): the only alignment a [T][Q] buffer with odd Q guarantees
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gmem_src) {
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
// wait until at most K of this thread's most recent groups are still in flight
template <int K>
__device__ __forceinline__ void cp_async_wait_group() { asm volatile("cp.async.wait_group %0;" ::"n"(K) : "memory"); }

// ---- mbarrier + TMA (bulk asynchronous copies: one instruction moves a whole tile / row, completion is counted in
// bytes on a shared-memory mbarrier; no per-thread LDGSTS, no L1TEX tag traffic)
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_init_fence() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// wait for the phase with the given parity to complete; gives up after ~2 s so a miscounted copy cannot hang the GPU
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    const unsigned a = smem_u32(bar);
    const long long t0 = clock64();
    for (;;) {
        unsigned ok;
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(a), "r"(parity) : "memory");
        if (ok) return;
        if (clock64() - t0 > 4000000000LL) { asm volatile("trap;"); }
    }
}
// generic-proxy accesses of shared memory that precede are ordered before asynchronous-proxy (TMA) accesses that follow
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// 2D tile of a tensor map -> shared memory (dense box), completion on `bar`
__device__ __forceinline__ void tma_load_2d(void* dst, const void* tmap, int c0, int c1, unsigned long long* bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(smem_u32(dst)), "l"(tmap), "r"(c0), "r"(c1), "r"(smem_u32(bar)) : "memory");
}
// contiguous bytes (multiple of 16, 16-byte aligned on both sides) -> shared memory, completion on `bar`
__device__ __forceinline__ void tma_load_1d(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// programmatic dependent launch: let the next kernel of the stream start launching / wait for the previous
// kernel of the stream to have completed (no-ops when the launch did not ask for it)
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

}  // namespace tacaw

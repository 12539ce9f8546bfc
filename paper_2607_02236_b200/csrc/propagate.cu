// propagate.cu -- the fused multislice slice step (K4) as two kernels per slice.
//
// The wave lives in the mixed (kx, y) layout W[y][kx] between kernels:
//   row kernel   (contiguous in kx):  W <- FFT_x{ t_{n+1} . IFFT_x{ W } }       (ROW_MID)
//   column kernel (stride nx):         W <- IFFT_y{ Px Py M/(nx ny) . FFT_y{ W } } (COL_MID)
// so one slice step  psi <- IFFT2{ P M FFT2{ t psi } }  (O5-O6) costs two read+write
// passes over the wave.  The band-limit mask makes columns |h| > hmax identically zero after the
// first step, so neither kernel touches them (2/3 of the traffic, 2/3 of the column FFTs).
// The Fresnel propagator is separable, P[h,k] = Px[h] Py[k]: two small tables, no HBM traffic.
// ROW_FIRST starts from the r-space entrance wave; ROW_LAST returns to r space; COL_LASTQ stops
// after the propagator multiply and stores the q-space exit wave Psi_S.  ROW_TRANS / COL_INV are
// the same transforms used by tacaw_build_slices and tacaw_make_probes.
#include <cstdlib>

#include "ctx.h"
#include "fft_core.cuh"

namespace tacaw {

// CTAs per launch aimed for (x SM count): a CTA loops over ceil(nwaves/chunks) waves, prefetching the
// next one while it transforms the current one.  TACAW_CTAS_PER_SM overrides (tuning only).
static int cta_target(const tacaw_ctx* ctx) {
    static int per_sm = [] {
        const char* e = getenv("TACAW_CTAS_PER_SM");
        int v = e ? atoi(e) : 0;
        return v > 0 ? v : 4;
    }();
    return ctx->num_sms * per_sm;
}

// ------------------------------------------------------------------------------------------
template <int N>
struct RowCfg {
    static constexpr int E = (N >= 1024) ? 16 : 8;
    static constexpr int T = N / E;
    static constexpr int THREADS = (T > 256) ? T : 256;   // upper bound on the CTA size
    static constexpr bool TWREG = (E == 8);
};

// Barrier functor that, the first time it fires after being armed, also issues the asynchronous
// prefetch of the next wave (every thread of the group has read the staging buffers by then).
template <class Base, class Issue>
struct SyncPrefetch {
    Base base;
    Issue issue;
    bool armed;
    __device__ __forceinline__ void operator()() {
        base();
        if (armed) {
            armed = false;
            issue();
        }
    }
};

template <int N, int MODE>
__global__ void __launch_bounds__(RowCfg<N>::THREADS) k_row(RowArgs a) {
    using C = RowCfg<N>;
    constexpr int E = C::E, T = C::T;
    constexpr bool TWREG = C::TWREG;
    constexpr bool HAS_T = (MODE == ROW_FIRST || MODE == ROW_MID);
    constexpr int XE = exch_elems(N, 1);
    constexpr int PER_G = 2 * XE + (HAS_T ? 2 : 1) * N;     // exchange A, exchange B, wave stage, t stage
    using P = FftPlan<N, E>;
    extern __shared__ __align__(16) float2 smem[];
    const int lt = threadIdx.x;
    const int g = lt / T, tid = lt % T;
    const int G = blockDim.x / T;
    const int row = blockIdx.x * G + g;
    float2* smA = smem + (size_t)g * PER_G;
    float2* smB = smA + XE;
    float2* sW = smA + 2 * XE;
    float2* sT = sW + N;
    const float2* roots_s = nullptr;
    float2 tw[P::NTW];
    if constexpr (TWREG) {
        TwInit<N, E, 1, 0>::run(tw, a.roots, tid);
    } else {
        float2* rs = smem + (size_t)G * PER_G;
        for (int i = lt; i < N; i += blockDim.x) rs[i] = a.roots[i];
        roots_s = rs;
        __syncthreads();
    }
    const int w0 = blockIdx.y * a.wpc;
    const int w1 = min(w0 + a.wpc, a.nwaves);
    const size_t npix = (size_t)a.ny * N;
    const size_t rowoff = (size_t)row * N;
    bool inb[E];
#pragma unroll
    for (int m = 0; m < E; ++m) {
        int ix = tid + T * m;
        inb[m] = (MODE == ROW_FIRST) || (ix <= a.hmax) || (ix >= N - a.hmax);
    }
    // asynchronous staging (LDGSTS, 16 B chunks): wave row -> sW (in-band chunks only), t row -> sT
    auto issue = [&](int w, bool with_t) {
        const float2* src;
        if constexpr (MODE == ROW_FIRST) src = a.probes ? a.probes + (size_t)a.wave_probe[w] * npix + rowoff
                                                        : a.waves + (size_t)w * npix + rowoff;
        else src = a.waves + (size_t)w * npix + rowoff;
#pragma unroll
        for (int j = 0; j < E / 2; ++j) {
            const int ix0 = 2 * (tid + T * j);
            const bool p = (MODE == ROW_FIRST) || (ix0 <= a.hmax) || (ix0 + 1 >= N - a.hmax);
            if (p) cp_async16(sW + ix0, src + ix0);
        }
        if constexpr (HAS_T) {
            if (with_t) {
                const float2* tp = a.trans[(size_t)a.wave_frame[w] * a.nseg + a.seg] + (size_t)a.slice * npix + rowoff;
#pragma unroll
                for (int j = 0; j < E / 2; ++j) {
                    const int ix0 = 2 * (tid + T * j);
                    cp_async16(sT + ix0, tp + ix0);
                }
            }
        }
        cp_async_commit();
    };
    auto body = [&](auto base_sync) {
        int cur_frame = -1;
        int next_w = w0;
        bool next_t = true;
        auto pf = [&]() { issue(next_w, next_t); };
        SyncPrefetch<decltype(base_sync), decltype(pf)> sync{base_sync, pf, false};
        if (w0 < w1) issue(w0, true);
        float2 tr[E];
        for (int w = w0; w < w1; ++w) {
            cp_async_wait_all();
            base_sync();
            float2 x[E];
#pragma unroll
            for (int m = 0; m < E; ++m) x[m] = inb[m] ? sW[tid + T * m] : make_float2(0.f, 0.f);
            if constexpr (HAS_T) {
                const int f = a.wave_frame[w];
                if (f != cur_frame) {
#pragma unroll
                    for (int m = 0; m < E; ++m) tr[m] = sT[tid + T * m];
                    cur_frame = f;
                }
            }
            if (w + 1 < w1) {
                next_w = w + 1;
                if constexpr (HAS_T) next_t = a.wave_frame[w + 1] != cur_frame;
                sync.armed = true;
            }
            float2* wrow = a.waves + (size_t)w * npix + rowoff;
            if constexpr (MODE != ROW_FIRST) {
                fft_regs<N, E, 1, true, TWREG, MODE == ROW_LAST>(x, tw, roots_s, smA, smB, tid, 0, sync);
                if constexpr (fft_nexch<N, E>() & 1) { float2* t_ = smA; smA = smB; smB = t_; }
            }
            if constexpr (HAS_T) {
#pragma unroll
                for (int m = 0; m < E; ++m) x[m] = cmul(x[m], tr[m]);
                fft_regs<N, E, 1, false, TWREG, true>(x, tw, roots_s, smA, smB, tid, 0, sync);
                if constexpr (fft_nexch<N, E>() & 1) { float2* t_ = smA; smA = smB; smB = t_; }
#pragma unroll
                for (int m = 0; m < E; ++m)
                    if (MODE == ROW_FIRST ? ((tid + T * m <= a.hmax) || (tid + T * m >= N - a.hmax)) : inb[m])
                        wrow[tid + T * m] = x[m];
            } else if constexpr (MODE == ROW_LAST) {
#pragma unroll
                for (int m = 0; m < E; ++m) wrow[tid + T * m] = x[m];
            } else {  // ROW_TRANS: t = exp(i sigma v), v = Re(x)/(lx ly)
#pragma unroll
                for (int m = 0; m < E; ++m) {
                    float s, c;
                    sincosf(a.scale * x[m].x, &s, &c);
                    wrow[tid + T * m] = make_float2(c, s);
                }
            }
        }
    };
    if constexpr (T <= 32) {
        body(SyncWarp{});
    } else {
        if (G == 1) body(SyncBlock{});
        else body(SyncNamed{1 + g, T});
    }
}

template <int N, int MODE>
static int launch_row_n(tacaw_ctx* ctx, const RowArgs& a0, cudaStream_t st) {
    using C = RowCfg<N>;
    RowArgs a = a0;
    int G = 256 / C::T;
    if (G < 1) G = 1;
    if (G > a.ny) G = a.ny;
    int threads = G * C::T;
    int nrb = a.ny / G;
    int target = cta_target(ctx);
    int nchunks = target / nrb;
    if (nchunks < 1) nchunks = 1;
    if (nchunks > a.nwaves) nchunks = a.nwaves;
    a.wpc = (a.nwaves + nchunks - 1) / nchunks;
    nchunks = (a.nwaves + a.wpc - 1) / a.wpc;
    const int per_g = 2 * exch_elems(N, 1) + ((MODE == ROW_FIRST || MODE == ROW_MID) ? 2 : 1) * N;
    size_t smem = (size_t)G * per_g * sizeof(float2) + (C::TWREG ? 0 : (size_t)N * sizeof(float2));
    auto kern = k_row<N, MODE>;
    if (smem > 48 * 1024) TACAW_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<dim3(nrb, nchunks), threads, smem, st>>>(a);
    ctx->launches++;
    TACAW_CUDA(ctx, cudaGetLastError());
    return TACAW_OK;
}

template <int N>
static int launch_row_mode(tacaw_ctx* ctx, int mode, const RowArgs& a, cudaStream_t st) {
    switch (mode) {
        case ROW_FIRST: return launch_row_n<N, ROW_FIRST>(ctx, a, st);
        case ROW_MID: return launch_row_n<N, ROW_MID>(ctx, a, st);
        case ROW_LAST: return launch_row_n<N, ROW_LAST>(ctx, a, st);
        case ROW_TRANS: return launch_row_n<N, ROW_TRANS>(ctx, a, st);
    }
    return fail(ctx, TACAW_E_ARG, "bad row mode");
}

int launch_row(tacaw_ctx* ctx, int mode, const RowArgs& a, cudaStream_t st) {
    if (a.nwaves <= 0) return TACAW_OK;
    switch (ctx->grid.nx) {
        case 16: return launch_row_mode<16>(ctx, mode, a, st);
        case 32: return launch_row_mode<32>(ctx, mode, a, st);
        case 64: return launch_row_mode<64>(ctx, mode, a, st);
        case 128: return launch_row_mode<128>(ctx, mode, a, st);
        case 256: return launch_row_mode<256>(ctx, mode, a, st);
        case 512: return launch_row_mode<512>(ctx, mode, a, st);
        case 1024: return launch_row_mode<1024>(ctx, mode, a, st);
        case 2048: return launch_row_mode<2048>(ctx, mode, a, st);
    }
    return fail(ctx, TACAW_E_UNSUPPORTED, "nx must be a power of two in [16, 2048]");
}

// ------------------------------------------------------------------------------------------
template <int N>
struct ColCfg {
    static constexpr int E = (N >= 1024) ? 16 : 8;
    static constexpr int T = N / E;
    static constexpr int WC = (N >= 512) ? 4 : 8;
    static constexpr int THREADS = T * WC;
    static constexpr bool TWREG = (E == 8);
};

template <int N, int MODE>
__global__ void __launch_bounds__(ColCfg<N>::THREADS) k_col(ColArgs a) {
    using C = ColCfg<N>;
    constexpr int E = C::E, T = C::T, WC = C::WC;
    constexpr bool TWREG = C::TWREG;
    using P = FftPlan<N, E>;
    extern __shared__ __align__(16) float2 smem[];
    const int lt = threadIdx.x;
    const int c = lt % WC, tid = lt / WC;
    constexpr int XE = exch_elems(N, WC);
    float2* smA = smem;
    float2* smB = smem + XE;
    const float2* roots_s = nullptr;
    // column group of this CTA
    const int NG = a.nx / WC;
    int grp = blockIdx.x;
    bool inband_group = true;
    {
        const int nlo = a.hmax / WC + 1;            // groups covering ix in [0, hmax]
        const int nhi = (a.hmax + WC - 1) / WC;     // groups covering ix in [nx-hmax, nx)
        if (a.all_groups) {
            inband_group = (nlo + nhi >= NG) || (grp < nlo) || (grp >= NG - nhi);
        } else if (nlo + nhi < NG) {
            grp = (grp < nlo) ? grp : NG - (nlo + nhi - grp);
        }
    }
    const int ix = grp * WC + c;
    const int w0 = blockIdx.y * a.wpc;
    const int w1 = min(w0 + a.wpc, a.nwaves);
    const size_t npix = (size_t)N * a.nx;

    if (MODE == COL_LASTQ && !inband_group) {       // out-of-band columns of Psi_S are exactly zero
        for (int w = w0; w < w1; ++w) {
            float2* wc = a.waves + (size_t)w * npix + ix;
#pragma unroll
            for (int m = 0; m < E; ++m) wc[(size_t)(tid + T * m) * a.nx] = make_float2(0.f, 0.f);
        }
        return;
    }

    float2* sW = smem + 2 * XE;                  // staging tile [N][WC]
    float2 tw[P::NTW];
    if constexpr (TWREG) {
        TwInit<N, E, 1, 0>::run(tw, a.roots, tid);
    } else {
        float2* rs = smem + 2 * XE + N * WC;
        for (int i = lt; i < N; i += blockDim.x) rs[i] = a.roots[i];
        roots_s = rs;
        __syncthreads();
    }
    float2 pxy[E];
    // a column that is entirely outside the mask is never written by the row kernel: do not use it
    // (it may hold anything, and NaN * 0 would not be 0)
    bool col_live = true;
    if constexpr (MODE != COL_INV) {
        const float2 px = a.px[ix];
        const int km = a.kmax[ix];
        col_live = km >= 0;
#pragma unroll
        for (int m = 0; m < E; ++m) {
            int ky = tid + T * m;
            int k = ky < N / 2 ? ky : N - ky;       // |k|
            float2 p = cmul(px, a.py[ky]);
            pxy[m] = (k <= km) ? make_float2(p.x * a.pscale, p.y * a.pscale) : make_float2(0.f, 0.f);
        }
    }
    // asynchronous staging of the [N][WC] tile of wave w: 16 B chunks, E/2 per thread
    auto issue = [&](int w) {
        const float2* src = a.waves + (size_t)w * npix + (size_t)grp * WC;
#pragma unroll
        for (int j = 0; j < E / 2; ++j) {
            const int id = lt + C::THREADS * j;
            const int r = id / (WC / 2), part = id % (WC / 2);
            cp_async16(sW + r * WC + 2 * part, src + (size_t)r * a.nx + 2 * part);
        }
        cp_async_commit();
    };
    auto body = [&](auto base_sync) {
        int next_w = w0;
        auto pf = [&]() { issue(next_w); };
        SyncPrefetch<decltype(base_sync), decltype(pf)> sync{base_sync, pf, false};
        if (w0 < w1) issue(w0);
        for (int w = w0; w < w1; ++w) {
            cp_async_wait_all();
            base_sync();
            float2* wc = a.waves + (size_t)w * npix + ix;
            float2 x[E];
#pragma unroll
            for (int m = 0; m < E; ++m) x[m] = col_live ? sW[(tid + T * m) * WC + c] : make_float2(0.f, 0.f);
            if (w + 1 < w1) {
                next_w = w + 1;
                sync.armed = true;
            }
            if constexpr (MODE != COL_INV) {
                fft_regs<N, E, WC, false, TWREG>(x, tw, roots_s, smA, smB, tid, c, sync);
                if constexpr (fft_nexch<N, E>() & 1) { float2* t_ = smA; smA = smB; smB = t_; }
#pragma unroll
                for (int m = 0; m < E; ++m) x[m] = cmul(x[m], pxy[m]);
            }
            if constexpr (MODE != COL_LASTQ) {
                fft_regs<N, E, WC, true, TWREG, true>(x, tw, roots_s, smA, smB, tid, c, sync);
                if constexpr (fft_nexch<N, E>() & 1) { float2* t_ = smA; smA = smB; smB = t_; }
            }
#pragma unroll
            for (int m = 0; m < E; ++m) wc[(size_t)(tid + T * m) * a.nx] = x[m];
        }
    };
    if constexpr (C::THREADS <= 32) body(SyncWarp{});
    else body(SyncBlock{});
}

template <int N, int MODE>
static int launch_col_n(tacaw_ctx* ctx, const ColArgs& a0, cudaStream_t st) {
    using C = ColCfg<N>;
    ColArgs a = a0;
    const int NG = a.nx / C::WC;
    int ngroups = NG;
    if (!a.all_groups) {
        int nlo = a.hmax / C::WC + 1, nhi = (a.hmax + C::WC - 1) / C::WC;
        if (nlo + nhi < NG) ngroups = nlo + nhi;
    }
    int target = cta_target(ctx);
    int nchunks = target / ngroups;
    if (nchunks < 1) nchunks = 1;
    if (nchunks > a.nwaves) nchunks = a.nwaves;
    a.wpc = (a.nwaves + nchunks - 1) / nchunks;
    nchunks = (a.nwaves + a.wpc - 1) / a.wpc;
    size_t smem = (size_t)(2 * exch_elems(N, C::WC) + N * C::WC) * sizeof(float2) + (C::TWREG ? 0 : (size_t)N * sizeof(float2));
    auto kern = k_col<N, MODE>;
    if (smem > 48 * 1024) TACAW_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<dim3(ngroups, nchunks), C::THREADS, smem, st>>>(a);
    ctx->launches++;
    TACAW_CUDA(ctx, cudaGetLastError());
    return TACAW_OK;
}

template <int N>
static int launch_col_mode(tacaw_ctx* ctx, int mode, const ColArgs& a, cudaStream_t st) {
    switch (mode) {
        case COL_MID: return launch_col_n<N, COL_MID>(ctx, a, st);
        case COL_LASTQ: return launch_col_n<N, COL_LASTQ>(ctx, a, st);
        case COL_INV: return launch_col_n<N, COL_INV>(ctx, a, st);
    }
    return fail(ctx, TACAW_E_ARG, "bad column mode");
}

int launch_col(tacaw_ctx* ctx, int mode, const ColArgs& a, int ny, cudaStream_t st) {
    if (a.nwaves <= 0) return TACAW_OK;
    switch (ny) {
        case 16: return launch_col_mode<16>(ctx, mode, a, st);
        case 32: return launch_col_mode<32>(ctx, mode, a, st);
        case 64: return launch_col_mode<64>(ctx, mode, a, st);
        case 128: return launch_col_mode<128>(ctx, mode, a, st);
        case 256: return launch_col_mode<256>(ctx, mode, a, st);
        case 512: return launch_col_mode<512>(ctx, mode, a, st);
        case 1024: return launch_col_mode<1024>(ctx, mode, a, st);
        case 2048: return launch_col_mode<2048>(ctx, mode, a, st);
    }
    return fail(ctx, TACAW_E_UNSUPPORTED, "ny must be a power of two in [16, 2048]");
}

}  // namespace tacaw

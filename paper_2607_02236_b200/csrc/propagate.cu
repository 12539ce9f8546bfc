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
#include "ctx.h"
#include "fft_core.cuh"

namespace tacaw {

// ------------------------------------------------------------------------------------------
template <int N>
struct RowCfg {
    static constexpr int E = (N >= 1024) ? 16 : 8;
    static constexpr int T = N / E;
    static constexpr int THREADS = (T > 256) ? T : 256;   // upper bound on the CTA size
    static constexpr bool TWREG = (E == 8);
};

template <int N, int MODE>
__global__ void __launch_bounds__(RowCfg<N>::THREADS) k_row(RowArgs a) {
    using C = RowCfg<N>;
    constexpr int E = C::E, T = C::T;
    constexpr bool TWREG = C::TWREG;
    using P = FftPlan<N, E>;
    extern __shared__ float2 smem[];
    const int lt = threadIdx.x;
    const int g = lt / T, tid = lt % T;
    const int G = blockDim.x / T;
    const int row = blockIdx.x * G + g;
    float2* smA = smem + (size_t)g * 2 * N;
    float2* smB = smA + N;
    const float2* roots_s = nullptr;
    float2 tw[P::NTW];
    if constexpr (TWREG) {
        TwInit<N, E, 1, 0>::run(tw, a.roots, tid);
    } else {
        float2* rs = smem + (size_t)G * 2 * N;
        for (int i = lt; i < N; i += blockDim.x) rs[i] = a.roots[i];
        roots_s = rs;
        __syncthreads();
    }
    auto body = [&](auto sync) {
        const int w0 = blockIdx.y * a.wpc;
        const int w1 = min(w0 + a.wpc, a.nwaves);
        const size_t npix = (size_t)a.ny * N;
        int cur_frame = -1;
        float2 tr[E];
        bool inb[E];
#pragma unroll
        for (int m = 0; m < E; ++m) {
            int ix = tid + T * m;
            inb[m] = (ix <= a.hmax) || (ix >= N - a.hmax);
        }
        for (int w = w0; w < w1; ++w) {
            float2 x[E];
            float2* wrow = a.waves + (size_t)w * npix + (size_t)row * N;
            if constexpr (MODE == ROW_FIRST || MODE == ROW_MID) {
                int f = a.wave_frame[w];
                if (f != cur_frame) {
                    const float2* tp = a.trans[(size_t)f * a.nseg + a.seg] + (size_t)a.slice * npix + (size_t)row * N;
#pragma unroll
                    for (int m = 0; m < E; ++m) tr[m] = __ldg(tp + tid + T * m);
                    cur_frame = f;
                }
            }
            if constexpr (MODE == ROW_FIRST) {
                const float2* src = a.probes ? a.probes + (size_t)a.wave_probe[w] * npix + (size_t)row * N : wrow;
#pragma unroll
                for (int m = 0; m < E; ++m) x[m] = src[tid + T * m];
            } else {
#pragma unroll
                for (int m = 0; m < E; ++m) x[m] = inb[m] ? wrow[tid + T * m] : make_float2(0.f, 0.f);
                fft_regs<N, E, 1, true, TWREG>(x, tw, roots_s, smA, smB, tid, 0, sync);
                if constexpr (fft_nexch<N, E>() & 1) { float2* t_ = smA; smA = smB; smB = t_; }
            }
            if constexpr (MODE == ROW_FIRST || MODE == ROW_MID) {
#pragma unroll
                for (int m = 0; m < E; ++m) x[m] = cmul(x[m], tr[m]);
                fft_regs<N, E, 1, false, TWREG>(x, tw, roots_s, smA, smB, tid, 0, sync);
                if constexpr (fft_nexch<N, E>() & 1) { float2* t_ = smA; smA = smB; smB = t_; }
#pragma unroll
                for (int m = 0; m < E; ++m)
                    if (inb[m]) wrow[tid + T * m] = x[m];
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
    int target = ctx->num_sms * 8;
    int nchunks = target / nrb;
    if (nchunks < 1) nchunks = 1;
    if (nchunks > a.nwaves) nchunks = a.nwaves;
    a.wpc = (a.nwaves + nchunks - 1) / nchunks;
    nchunks = (a.nwaves + a.wpc - 1) / a.wpc;
    size_t smem = (size_t)G * 2 * N * sizeof(float2) + (C::TWREG ? 0 : (size_t)N * sizeof(float2));
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
    extern __shared__ float2 smem[];
    const int lt = threadIdx.x;
    const int c = lt % WC, tid = lt / WC;
    float2* smA = smem;
    float2* smB = smem + (size_t)N * WC;
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

    float2 tw[P::NTW];
    if constexpr (TWREG) {
        TwInit<N, E, 1, 0>::run(tw, a.roots, tid);
    } else {
        float2* rs = smem + (size_t)2 * N * WC;
        for (int i = lt; i < N; i += blockDim.x) rs[i] = a.roots[i];
        roots_s = rs;
        __syncthreads();
    }
    float2 pxy[E];
    // a column that is entirely outside the mask is never written by the row kernel: do not read it
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
    auto body = [&](auto sync) {
        for (int w = w0; w < w1; ++w) {
            float2* wc = a.waves + (size_t)w * npix + ix;
            float2 x[E];
#pragma unroll
            for (int m = 0; m < E; ++m) x[m] = col_live ? wc[(size_t)(tid + T * m) * a.nx] : make_float2(0.f, 0.f);
            if constexpr (MODE != COL_INV) {
                fft_regs<N, E, WC, false, TWREG>(x, tw, roots_s, smA, smB, tid, c, sync);
                if constexpr (fft_nexch<N, E>() & 1) { float2* t_ = smA; smA = smB; smB = t_; }
#pragma unroll
                for (int m = 0; m < E; ++m) x[m] = cmul(x[m], pxy[m]);
            }
            if constexpr (MODE != COL_LASTQ) {
                fft_regs<N, E, WC, true, TWREG>(x, tw, roots_s, smA, smB, tid, c, sync);
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
    int target = ctx->num_sms * 8;
    int nchunks = target / ngroups;
    if (nchunks < 1) nchunks = 1;
    if (nchunks > a.nwaves) nchunks = a.nwaves;
    a.wpc = (a.nwaves + nchunks - 1) / nchunks;
    nchunks = (a.nwaves + a.wpc - 1) / a.wpc;
    size_t smem = (size_t)2 * N * C::WC * sizeof(float2) + (C::TWREG ? 0 : (size_t)N * sizeof(float2));
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

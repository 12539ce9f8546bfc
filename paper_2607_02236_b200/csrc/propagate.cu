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

// ------------------------------------------------------------------------------------------
template <int N>
struct RowCfg {
    static constexpr int E = (N >= 1024) ? 16 : 8;
    static constexpr int T = N / E;
    static constexpr int THREADS = (T > 256) ? T : 256;   // upper bound on the CTA size
    static constexpr bool TWREG = (E == 8);
    static constexpr int MINB = (E == 8) ? 3 : 1;          // CTAs per SM the register budget is held to
};

// Barrier functor that, the first time it fires after being armed, also issues the asynchronous
// prefetch of the next work item (every thread of the group has read the staging buffers by then).
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

// Work items of a row launch are (row block, wave) pairs, flattened as rb*nwaves + w and dealt out
// in equal contiguous ranges to a grid that exactly fills the machine (no partial last wave of
// CTAs).  Consecutive items of a CTA share the row block, so the t_n row is reloaded only when the
// frame (or the row block) changes.
template <int N, int MODE>
__global__ void __launch_bounds__(RowCfg<N>::THREADS, RowCfg<N>::MINB) k_row(RowArgs a) {
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
    const long long i0 = (long long)blockIdx.x * a.ipc;
    const long long i1 = min(i0 + (long long)a.ipc, a.nitems);
    const size_t npix = (size_t)a.ny * N;
    bool inb[E];
#pragma unroll
    for (int m = 0; m < E; ++m) {
        int ix = tid + T * m;
        inb[m] = (MODE == ROW_FIRST) || (ix <= a.hmax) || (ix >= N - a.hmax);
    }
    // asynchronous staging (LDGSTS, 16 B chunks): wave row -> sW (in-band chunks only), t row -> sT
    auto issue_wave = [&](int w, size_t rowoff) {
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
    };
    auto issue_t = [&](int f, size_t rowoff) {
        const float2* tp = a.trans[(size_t)f * a.nseg + a.seg] + (size_t)a.slice * npix + rowoff;
#pragma unroll
        for (int j = 0; j < E / 2; ++j) {
            const int ix0 = 2 * (tid + T * j);
            cp_async16(sT + ix0, tp + ix0);
        }
    };
    auto body = [&](auto base_sync) {
        int cur_frame = -1, cur_rb = -1;
        int next_w = 0, next_f = -1;
        size_t next_rowoff = 0;
        int phase = 0;      // which prefetch the next barrier hook issues: 0 wave row, 1 t row
        auto pf = [&]() {
            if (phase == 0) issue_wave(next_w, next_rowoff);
            if constexpr (HAS_T) {
                if ((phase == 1 || MODE == ROW_FIRST) && next_f >= 0) issue_t(next_f, next_rowoff);
            }
            cp_async_commit();
        };
        SyncPrefetch<decltype(base_sync), decltype(pf)> sync{base_sync, pf, false};
        if (i0 < i1) {
            const int rb = (int)(i0 / a.nwaves), w = (int)(i0 - (long long)rb * a.nwaves);
            const size_t rowoff = (size_t)(rb * G + g) * N;
            issue_wave(w, rowoff);
            if constexpr (HAS_T) {
                cur_frame = a.wave_frame[w];
                cur_rb = rb;
                issue_t(cur_frame, rowoff);
            }
            cp_async_commit();
        }
        for (long long i = i0; i < i1; ++i) {
            const int rb = (int)(i / a.nwaves), w = (int)(i - (long long)rb * a.nwaves);
            const size_t rowoff = (size_t)(rb * G + g) * N;
            cp_async_wait_all();
            base_sync();
            float2 x[E];
#pragma unroll
            for (int m = 0; m < E; ++m) x[m] = inb[m] ? sW[tid + T * m] : make_float2(0.f, 0.f);
            const bool more = (i + 1 < i1);
            next_f = -1;
            if (more) {
                const int rbn = (int)((i + 1) / a.nwaves);
                next_w = (int)(i + 1 - (long long)rbn * a.nwaves);
                next_rowoff = (size_t)(rbn * G + g) * N;
                if constexpr (HAS_T) {
                    const int f = a.wave_frame[next_w];
                    if (f != cur_frame || rbn != cur_rb) { next_f = f; cur_frame = f; cur_rb = rbn; }
                }
            }
            float2* wrow = a.waves + (size_t)w * npix + rowoff;
            if constexpr (MODE != ROW_FIRST) {
                phase = 0;
                sync.armed = more;
                fft_regs<N, E, 1, true, TWREG, MODE == ROW_LAST>(x, tw, roots_s, smA, smB, tid, 0, sync);
                if constexpr (fft_nexch<N, E>() & 1) { float2* t_ = smA; smA = smB; smB = t_; }
            }
            if constexpr (HAS_T) {
                // t_n row from the staging buffer; its successor is prefetched only after this use
#pragma unroll
                for (int m = 0; m < E; ++m) x[m] = cmul(x[m], sT[tid + T * m]);
                if constexpr (MODE == ROW_FIRST) { phase = 0; sync.armed = more; }
                else { phase = 1; sync.armed = (next_f >= 0); }
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

// grid that fills the machine exactly: occupancy x SM count CTAs (or one CTA per item if fewer)
template <class K>
static int machine_ctas(const tacaw_ctx* ctx, K kern, int threads, size_t smem, int* cache) {
    if (*cache == 0) {
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, smem) != cudaSuccess || per_sm < 1) {
            (void)cudaGetLastError();
            per_sm = 1;
        }
        *cache = per_sm;
    }
    return ctx->num_sms * (*cache);
}

template <int N, int MODE>
static int launch_row_n(tacaw_ctx* ctx, const RowArgs& a0, cudaStream_t st) {
    using C = RowCfg<N>;
    RowArgs a = a0;
    int G = 256 / C::T;
    if (G < 1) G = 1;
    if (G > a.ny) G = a.ny;
    const int threads = G * C::T;
    const int nrb = a.ny / G;
    const int per_g = 2 * exch_elems(N, 1) + ((MODE == ROW_FIRST || MODE == ROW_MID) ? 2 : 1) * N;
    const size_t smem = (size_t)G * per_g * sizeof(float2) + (C::TWREG ? 0 : (size_t)N * sizeof(float2));
    auto kern = k_row<N, MODE>;
    static bool attr_set = false;
    if (!attr_set) {
        if (smem > 48 * 1024) TACAW_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_set = true;
    }
    static int occ_cache[4] = {0, 0, 0, 0};     // per CTA size class (G varies only for tiny ny)
    int* cache = &occ_cache[threads == 256 ? 0 : (threads == 128 ? 1 : (threads == 64 ? 2 : 3))];
    if (threads != 256 && threads != 128 && threads != 64) *cache = 0;
    a.nitems = (long long)nrb * a.nwaves;
    long long ctas = machine_ctas(ctx, kern, threads, smem, cache);
    if (ctas > a.nitems) ctas = a.nitems;
    a.ipc = (int)((a.nitems + ctas - 1) / ctas);
    ctas = (a.nitems + a.ipc - 1) / a.ipc;
    kern<<<(unsigned)ctas, threads, smem, st>>>(a);
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
    static constexpr bool USE_SP = (E == 8);     // propagator factors in shared memory instead of registers
    static constexpr int MINB = (E == 8 && THREADS <= 256) ? 3 : 1;
};

// Work items of a column launch are (column group, wave) pairs, flattened as gi*nwaves + w over the
// selected groups (the in-band ones, or all of them when hmax covers the grid) and dealt out in equal
// contiguous ranges to a machine-filling grid, like the row kernel.
template <int N, int MODE>
__global__ void __launch_bounds__(ColCfg<N>::THREADS, ColCfg<N>::MINB) k_col(ColArgs a) {
    using C = ColCfg<N>;
    constexpr int E = C::E, T = C::T, WC = C::WC;
    constexpr bool TWREG = C::TWREG, USE_SP = C::USE_SP && (MODE != COL_INV);
    using P = FftPlan<N, E>;
    extern __shared__ __align__(16) float2 smem[];
    const int lt = threadIdx.x;
    const int c = lt % WC, tid = lt / WC;
    constexpr int XE = exch_elems(N, WC);
    float2* smA = smem;
    float2* smB = smem + XE;
    float2* sW = smem + 2 * XE;                  // staging tile [N][WC]
    float2* sP = sW + N * WC;                    // Px Py M /(nx ny) of this CTA's column group (USE_SP)
    const float2* roots_s = nullptr;
    float2 tw[P::NTW];
    if constexpr (TWREG) {
        TwInit<N, E, 1, 0>::run(tw, a.roots, tid);
    } else {
        float2* rs = sW + N * WC + (C::USE_SP ? N * WC : 0);
        for (int i = lt; i < N; i += blockDim.x) rs[i] = a.roots[i];
        roots_s = rs;
        __syncthreads();
    }
    const int NG = a.nx / WC;
    const int nlo = a.hmax / WC + 1;            // groups covering ix in [0, hmax]
    const int nhi = (a.hmax + WC - 1) / WC;     // groups covering ix in [nx-hmax, nx)
    const bool all = (nlo + nhi >= NG);
    auto group_of = [&](int gi) { return (all || gi < nlo) ? gi : NG - (nlo + nhi - gi); };
    const long long i0 = (long long)blockIdx.x * a.ipc;
    const long long i1 = min(i0 + (long long)a.ipc, a.nitems);
    const size_t npix = (size_t)N * a.nx;

    float2 pxy[C::USE_SP ? 1 : E];
    bool col_live = true;
    int cur_grp = -1;
    // propagator factors of column ix: Px[h] Py[k] M[h,k] pscale.  A column that is entirely outside
    // the mask is never written by the row kernel: it is not used (NaN * 0 would not be 0).
    auto load_factors = [&](int grp) {
        if constexpr (MODE != COL_INV) {
            const int ix = grp * WC + c;
            const float2 px = a.px[ix];
            const int km = a.kmax[ix];
            col_live = km >= 0;
#pragma unroll
            for (int m = 0; m < E; ++m) {
                int ky = tid + T * m;
                int k = ky < N / 2 ? ky : N - ky;       // |k|
                float2 p = cmul(px, a.py[ky]);
                float2 v = (k <= km) ? make_float2(p.x * a.pscale, p.y * a.pscale) : make_float2(0.f, 0.f);
                if constexpr (USE_SP) sP[ky * WC + c] = v;      // thread-private slot
                else pxy[m] = v;
            }
        }
    };
    // asynchronous staging of the [N][WC] tile of wave w: 16 B chunks, E/2 per thread
    auto issue = [&](int w, int grp) {
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
        int next_w = 0, next_grp = 0;
        auto pf = [&]() { issue(next_w, next_grp); };
        SyncPrefetch<decltype(base_sync), decltype(pf)> sync{base_sync, pf, false};
        if (i0 < i1) {
            const int gi = (int)(i0 / a.nwaves);
            issue((int)(i0 - (long long)gi * a.nwaves), group_of(gi));
        }
        for (long long i = i0; i < i1; ++i) {
            const int gi = (int)(i / a.nwaves), w = (int)(i - (long long)gi * a.nwaves);
            const int grp = group_of(gi);
            if (grp != cur_grp) { load_factors(grp); cur_grp = grp; }
            cp_async_wait_all();
            base_sync();
            float2* wc = a.waves + (size_t)w * npix + (size_t)grp * WC + c;
            float2 x[E];
#pragma unroll
            for (int m = 0; m < E; ++m) x[m] = col_live ? sW[(tid + T * m) * WC + c] : make_float2(0.f, 0.f);
            if (i + 1 < i1) {
                const int gn = (int)((i + 1) / a.nwaves);
                next_w = (int)(i + 1 - (long long)gn * a.nwaves);
                next_grp = group_of(gn);
                sync.armed = true;
            }
            if constexpr (MODE != COL_INV) {
                fft_regs<N, E, WC, false, TWREG>(x, tw, roots_s, smA, smB, tid, c, sync);
                if constexpr (fft_nexch<N, E>() & 1) { float2* t_ = smA; smA = smB; smB = t_; }
#pragma unroll
                for (int m = 0; m < E; ++m) {
                    if constexpr (USE_SP) x[m] = cmul(x[m], sP[(tid + T * m) * WC + c]);
                    else x[m] = cmul(x[m], pxy[m]);
                }
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

// zero the out-of-band columns [c0, c1) of every row of every wave (exit wave Psi_S, O7)
__global__ void k_zero_cols(float2* __restrict__ waves, long long nrows, int nx, int c0, int c1) {
    const int width = (c1 - c0) / 2;      // float4 = two complex values; c0, c1 are even
    const long long total = nrows * width;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const long long r = i / width;
        const int j = (int)(i - r * width);
        reinterpret_cast<float4*>(waves + r * nx + c0)[j] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
}

template <int N, int MODE>
static int launch_col_n(tacaw_ctx* ctx, const ColArgs& a0, cudaStream_t st) {
    using C = ColCfg<N>;
    ColArgs a = a0;
    const int NG = a.nx / C::WC;
    const int nlo = a.hmax / C::WC + 1, nhi = (a.hmax + C::WC - 1) / C::WC;
    const bool all = nlo + nhi >= NG;
    const int ngroups = all ? NG : nlo + nhi;
    const size_t smem = (size_t)(2 * exch_elems(N, C::WC) + (C::USE_SP ? 2 : 1) * N * C::WC) * sizeof(float2) +
                        (C::TWREG ? 0 : (size_t)N * sizeof(float2));
    auto kern = k_col<N, MODE>;
    static bool attr_set = false;
    if (!attr_set) {
        if (smem > 48 * 1024) TACAW_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_set = true;
    }
    static int occ_cache = 0;
    a.nitems = (long long)ngroups * a.nwaves;
    long long ctas = machine_ctas(ctx, kern, C::THREADS, smem, &occ_cache);
    if (ctas > a.nitems) ctas = a.nitems;
    a.ipc = (int)((a.nitems + ctas - 1) / ctas);
    ctas = (a.nitems + a.ipc - 1) / a.ipc;
    kern<<<(unsigned)ctas, C::THREADS, smem, st>>>(a);
    ctx->launches++;
    if (MODE == COL_LASTQ && !all) {
        const int c0 = nlo * C::WC, c1 = (NG - nhi) * C::WC;
        const long long nrows = (long long)a.nwaves * N;
        long long blocks = (nrows * ((c1 - c0) / 2) + 255) / 256;
        if (blocks > ctx->num_sms * 16) blocks = ctx->num_sms * 16;
        k_zero_cols<<<(unsigned)blocks, 256, 0, st>>>(a.waves, nrows, a.nx, c0, c1);
        ctx->launches++;
    }
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

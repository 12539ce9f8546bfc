// spectrum.cu -- K6: window x batched time FFT x |.|^2 x Bose/detailed-balance factor.
//
//   Phi_k = sum_f w_f buf[p][f][r] exp(-2 pi i k f/T)                     (O9, O10)
//   I[p][e][r] = B(E_e/kBT) |Phi_k|^2 / (T sum w^2),  energies ascending, cropped to the E-ROI
// buf is [P][T][Q] (r fastest), so a CTA takes a [T x WQ] tile -- the same vector-FFT machinery as
// the multislice column kernel: thread (tid, c) holds frames tid + Tt*m of series r0+c, the
// transform leaves it with bins tid + Tt*m, which it scales and stores.  The window and the
// per-energy factor bose[e] = B(E_e/kBT)/(T sum w^2) are fp64-computed host tables.
#include <cstdlib>

#include "ctx.h"
#include "fft2.cuh"

namespace tacaw {

template <int N>
struct SpecCfg {
    static constexpr int E = (N >= 1024) ? 16 : 8;
    static constexpr int T = N / E;
    // series per CTA: 128-byte (64-byte at 512) row segments of the [T][Q] buffer where the tile still leaves several CTAs
    // per SM (measured: T=256 0.077 -> 0.072 ms, T=512 0.90 -> 0.72 ms for 32 x 7721 series; wider tiles at 1024 were slower)
    static constexpr int WQ = (N <= 256) ? 16 : ((N <= 512) ? 8 : 4);
    static constexpr int THREADS = T * WQ;
    static constexpr bool TWREG = (E == 8);
};

template <int N>
__global__ void __launch_bounds__(SpecCfg<N>::THREADS) k_spectrum(const float2* __restrict__ buf, long long nroi,
                                                                  size_t probe_stride, size_t frame_stride, int nchunks,
                                                                  size_t chunk_stride, const float2* __restrict__ roots,
                                                                  const float* __restrict__ window,
                                                                  const float* __restrict__ bose, int e_lo, int nE,
                                                                  float* __restrict__ I) {
    using C = SpecCfg<N>;
    constexpr int E = C::E, T = C::T, WQ = C::WQ;
    constexpr bool TWREG = C::TWREG;
    using P = FftPlan<N, E>;
    extern __shared__ __align__(16) float2 smem[];
    const int lt = threadIdx.x;
    const int c = lt % WQ, tid = lt / WQ;
    constexpr int XE = exch_elems(N, WQ);
    float2* smA = smem;
    float2* smB = smem + XE;
    const float2* roots_s = nullptr;
    float2 tw[P::NTW];
    if constexpr (TWREG) {
        TwInit<N, E, 1, 0>::run(tw, roots, tid);
    } else {
        float2* rs = smem + 2 * XE;
        for (int i = lt; i < N; i += blockDim.x) rs[i] = roots[i];
        roots_s = rs;
        __syncthreads();
    }
    const int p = blockIdx.y;
    const long long r = (long long)blockIdx.x * WQ + c;
    const bool live = r < nroi;
    const float2* src = buf + (size_t)p * probe_stride + (live ? r : 0);
    // Welch chunks (Eq.(2)): every chunk of the series is transformed here and |Phi|^2 summed in registers, so I is
    // written once (bose[] carries the 1/N of the average)
    float acc[E];
#pragma unroll
    for (int m = 0; m < E; ++m) acc[m] = 0.f;
    for (int ch = 0; ch < nchunks; ++ch, src += chunk_stride) {
        float2 x[E];
#pragma unroll
        for (int m = 0; m < E; ++m) {
            int f = tid + T * m;
            float2 v = live ? src[(size_t)f * frame_stride] : make_float2(0.f, 0.f);
            float w = window[f];
            x[m] = make_float2(v.x * w, v.y * w);
        }
        if constexpr (C::THREADS <= 32) {
            SyncWarp sync;
            if (ch > 0) sync();
            fft_regs<N, E, WQ, false, TWREG>(x, tw, roots_s, smA, smB, tid, c, sync);
        } else {
            SyncBlock sync;
            if (ch > 0) sync();                         // the previous chunk's last exchange has been read back
            fft_regs<N, E, WQ, false, TWREG>(x, tw, roots_s, smA, smB, tid, c, sync);
        }
#pragma unroll
        for (int m = 0; m < E; ++m) acc[m] += x[m].x * x[m].x + x[m].y * x[m].y;
    }
    if (!live) return;
    float* dst = I + (size_t)p * nE * (size_t)nroi + r;
#pragma unroll
    for (int m = 0; m < E; ++m) {
        int kbin = tid + T * m;
        int e = ((kbin + N / 2) & (N - 1)) - e_lo;      // position on the ascending energy axis
        if (e >= 0 && e < nE) dst[(size_t)e * nroi] = bose[e] * acc[m];
    }
}

// Series of 512 frames and more: the single-exchange transform of the slice-step kernels (fft2.cuh; thread (tid, c) holds the
// 32 frames tid + Tt*m of series r0+c, one padded exchange, twiddles from the Plan2 table in shared memory).  Half the
// shared memory of the ping-pong plan above and twice the loads in flight per thread.
template <int N>
struct SpecCfg2 {
    using P = Plan2<N>;
    static constexpr int E = P::E, T = P::T;
    // series per CTA, measured on B200 for 32 x 7721 series (ms at 512 / 1024 / 2048 frames): 8: 0.69 / 1.52 / 3.37,
    // 16: 0.63 / 1.60 / -, 4: - / 1.95 / 3.87; the two-exchange plan above: 0.75 / 1.83 / 4.28
    static constexpr int WQ = (N == 512) ? 16 : 8;
    static constexpr int THREADS = T * WQ;
    static constexpr int XE = exch2_elems(N, WQ);
    // twiddles | exchange / staging tile | window [N] | Bose factors of the kept bins [<= N]
    static constexpr size_t smem() { return sizeof(float2) * ((size_t)P::TW_ELEMS + XE) + sizeof(float) * 2 * N; }
    static_assert(P::TW_ELEMS % 2 == 0 && XE % 2 == 0, "16-byte alignment of the staging tile and of the float tables");
};

// Persistent: a CTA walks (tile, chunk) work items with stride gridDim.x.  The [T][WQ] tile of the NEXT item is requested
// with 8-byte cp.async copies into the exchange buffer as soon as the exchange of the current item has been read back (the
// buffer is idle during the second radix pass, |.|^2 and the stores), so the strided global reads of one item overlap the
// arithmetic of the previous one instead of heading every item (round 1: one tile per CTA, DRAM 23 % busy, every warp
// waiting on its own 32 loads).
// WELCH = false (one chunk): no accumulator registers, |Phi|^2 goes straight to the store.
template <int N, bool WELCH>
__global__ void __launch_bounds__(SpecCfg2<N>::THREADS, (SpecCfg2<N>::THREADS >= 512 ? 1 : 2)) k_spectrum2(const float2* __restrict__ buf, long long nroi, int nprobes,
                                                                    size_t probe_stride, size_t frame_stride, int nchunks,
                                                                    size_t chunk_stride, const float2* __restrict__ table,
                                                                    const float* __restrict__ window,
                                                                    const float* __restrict__ bose, int e_lo, int nE,
                                                                    float* __restrict__ I) {
    using C = SpecCfg2<N>;
    using P = Plan2<N>;
    constexpr int E = C::E, T = C::T, WQ = C::WQ;
    extern __shared__ __align__(16) float2 smem[];
    const int lt = threadIdx.x;
    const int c = lt % WQ, tid = lt / WQ;
    float2* tw = smem;
    float2* ex = smem + P::TW_ELEMS;
    float* sw = reinterpret_cast<float*>(ex + C::XE);             // window and Bose tables: read by every item of this CTA
    float* sb = sw + N;
    fft2_load_twiddles<N>(tw, table, lt, C::THREADS);
    for (int i = lt; i < N; i += C::THREADS) {
        sw[i] = window[i];
        sb[i] = i < nE ? bose[i] : 0.f;
    }
    // even Q (and even strides): a row segment of the tile is 16-byte aligned, so two series go per cp.async
    const bool vec2 = ((nroi | (long long)probe_stride | (long long)frame_stride | (long long)chunk_stride) & 1) == 0 &&
                      (reinterpret_cast<uintptr_t>(buf) & 15) == 0;
    const long long ntq = (nroi + WQ - 1) / WQ;
    const long long ntiles = ntq * nprobes;                    // tile = (probe, q tile); a CTA takes tiles blockIdx.x + k gridDim.x
    auto issue = [&](long long tile, int ch) {                 // and runs all chunks of a tile before the next tile
        const int p = (int)(tile / ntq);
        const long long r = (tile - (long long)p * ntq) * WQ + c;
        const float2* src = buf + (size_t)p * probe_stride + (size_t)ch * chunk_stride + r;
        if (vec2) {
            const int c2 = 2 * (lt % (WQ / 2)), rb = lt / (WQ / 2);         // series pair, first of this thread's E/2 rows
            const long long r2 = r - c + c2;
            const float2* src2 = src - c + c2;
            if (r2 < nroi) {
#pragma unroll
                for (int j = 0; j < E / 2; ++j) cp_async16(ex + (rb + 2 * T * j) * WQ + c2, src2 + (size_t)(rb + 2 * T * j) * frame_stride);
            } else {
#pragma unroll
                for (int j = 0; j < E / 2; ++j) {
                    ex[(rb + 2 * T * j) * WQ + c2] = make_float2(0.f, 0.f);
                    ex[(rb + 2 * T * j) * WQ + c2 + 1] = make_float2(0.f, 0.f);
                }
            }
        } else if (r < nroi) {
#pragma unroll
            for (int m = 0; m < E; ++m) cp_async8(ex + (tid + T * m) * WQ + c, src + (size_t)(tid + T * m) * frame_stride);
        } else {
#pragma unroll
            for (int m = 0; m < E; ++m) ex[(tid + T * m) * WQ + c] = make_float2(0.f, 0.f);
        }
        cp_async_commit();
    };
    long long tile = blockIdx.x;
    int ch = 0;
    if (tile < ntiles) issue(tile, 0);
    float acc[WELCH ? E : 1];                      // sum over the Welch chunks of |Phi|^2 (Eq.(2)); I is written once per tile
    SyncBlock sync;
    while (tile < ntiles) {
        if constexpr (WELCH) {
            if (ch == 0) {
#pragma unroll
                for (int m = 0; m < E; ++m) acc[m] = 0.f;
            }
        }
        cp_async_wait_all();
        __syncthreads();                           // tile (and, the first time, the twiddle table) complete
        float2 x[E];
#pragma unroll
        for (int m = 0; m < E; ++m) {
            const float2 v = ex[(tid + T * m) * WQ + c];
            const float wm = sw[tid + T * m];
            x[m] = make_float2(v.x * wm, v.y * wm);
        }
        __syncthreads();                           // tile consumed: the exchange may overwrite it
        const bool last_ch = (ch == nchunks - 1);
        const long long ntile = last_ch ? tile + gridDim.x : tile;
        const int nch = last_ch ? 0 : ch + 1;
        auto nopre = []() {};
        auto post = [&]() {
            if (ntile < ntiles) {
                __syncthreads();                   // exchange read back by every thread
                issue(ntile, nch);
            }
        };
        Hooks<decltype(nopre), decltype(post)> hook{nopre, post};
        fft2<N, WQ, false, false>(x, tw + tid, ex, tid, c, sync, hook);
        if constexpr (WELCH) {
#pragma unroll
            for (int m = 0; m < E; ++m) acc[m] += x[m].x * x[m].x + x[m].y * x[m].y;
        }
        if (last_ch) {
            const int p = (int)(tile / ntq);
            const long long r = (tile - (long long)p * ntq) * WQ + c;
            if (r < nroi) {
                float* dst = I + (size_t)p * nE * (size_t)nroi + r;
#pragma unroll
                for (int m = 0; m < E; ++m) {
                    const int kbin = tid + T * m;
                    const int e = ((kbin + N / 2) & (N - 1)) - e_lo;      // position on the ascending energy axis
                    if (e >= 0 && e < nE) dst[(size_t)e * nroi] = sb[e] * (WELCH ? acc[m] : x[m].x * x[m].x + x[m].y * x[m].y);
                }
            }
        }
        tile = ntile;
        ch = nch;
    }
    cp_async_wait_all();
}

template <int N>
static int launch_spec2_n(tacaw_ctx* ctx, const float2* d_buf, int nprobes, int64_t nroi, size_t probe_stride, size_t frame_stride,
                          int nchunks, size_t chunk_stride, const float2* table,
                          const float* d_window, const float* d_bose, int e_lo, int nE, float* d_I,
                          cudaStream_t st) {
    using C = SpecCfg2<N>;
    const size_t smem = C::smem();
    auto kern = nchunks > 1 ? k_spectrum2<N, true> : k_spectrum2<N, false>;
    const void* key = (const void*)kern;
    auto itc = ctx->kernel_occ.find(key);
    if (itc == ctx->kernel_occ.end()) {
        if (smem > 48 * 1024) TACAW_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, C::THREADS, smem) != cudaSuccess || per_sm < 1) {
            (void)cudaGetLastError();
            per_sm = 1;
        }
        itc = ctx->kernel_occ.emplace(key, per_sm).first;
    }
    const long long ntiles = ((nroi + C::WQ - 1) / C::WQ) * (long long)nprobes;
    long long grid = (long long)ctx->num_sms * itc->second;
    if (grid > ntiles) grid = ntiles;
    if (grid > 0) {
        kern<<<(unsigned)grid, C::THREADS, smem, st>>>(d_buf, (long long)nroi, nprobes, probe_stride, frame_stride, nchunks, chunk_stride, table,
                                                     d_window, d_bose, e_lo, nE, d_I);
        ctx->launches++;
    }
    TACAW_CUDA(ctx, cudaGetLastError());
    return TACAW_OK;
}

template <int N>
static int launch_spec_n(tacaw_ctx* ctx, const float2* d_buf, int nprobes, int64_t nroi, size_t probe_stride, size_t frame_stride,
                         int nchunks, size_t chunk_stride, const float2* roots,
                         const float* d_window, const float* d_bose, int e_lo, int nE, float* d_I, cudaStream_t st) {
    using C = SpecCfg<N>;
    size_t smem = (size_t)2 * exch_elems(N, C::WQ) * sizeof(float2) + (C::TWREG ? 0 : (size_t)N * sizeof(float2));
    auto kern = k_spectrum<N>;
    if (smem > 48 * 1024) TACAW_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int64_t gx = (nroi + C::WQ - 1) / C::WQ;
    for (int p0 = 0; p0 < nprobes; p0 += 32768) {
        int np = nprobes - p0 < 32768 ? nprobes - p0 : 32768;
        kern<<<dim3((unsigned)gx, np), C::THREADS, smem, st>>>(d_buf + (size_t)p0 * probe_stride, (long long)nroi, probe_stride, frame_stride,
                                                              nchunks, chunk_stride, roots, d_window, d_bose, e_lo, nE,
                                                              d_I + (size_t)p0 * nE * (size_t)nroi);
        ctx->launches++;
    }
    TACAW_CUDA(ctx, cudaGetLastError());
    return TACAW_OK;
}

// Series of any other length (the paper's default chunk of 200 snapshots, Listing 1 :442): the time transform as
// the plain DFT sum restricted to the energy ROI,  Phi_e = sum_f W[e][f] x[f],  W[e][f] = w_f exp(-2 pi i k_e f/L) (host table,
// fp64 with the phase index k_e f mod L reduced exactly).  A CTA holds a [L x 32 series] tile in shared memory; a warp owns
// every fourth group of four energies and keeps their four sums in registers, one series per lane (coalesced loads of the
// buffer, broadcast reads of W).  Work is nE L complex multiply-adds per series -- the spectrum is a small share of the path
// and with an energy ROI only the wanted bins are computed.
constexpr int DFT_SER = 32;        // series per CTA
constexpr int DFT_WARPS = 4;
constexpr int DFT_EB = 4;          // energies per register block

__global__ void __launch_bounds__(DFT_SER * DFT_WARPS) k_spectrum_dft(const float2* __restrict__ buf, long long nroi, size_t probe_stride,
                                                                      size_t frame_stride, int nchunks, size_t chunk_stride, int L,
                                                                      const float2* __restrict__ W, const float* __restrict__ bose,
                                                                      int nE, float* __restrict__ I) {
    extern __shared__ __align__(16) float2 xs[];          // [L][DFT_SER] tile of the chunk, then [nE][DFT_SER] sums of |Phi|^2
    float* accs = reinterpret_cast<float*>(xs + (size_t)L * DFT_SER);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int p = blockIdx.y;
    const long long r = (long long)blockIdx.x * DFT_SER + lane;
    const bool live = r < nroi;
    const float2* src = buf + (size_t)p * probe_stride + (live ? r : 0);
    for (int e0 = warp * DFT_EB; e0 < nE; e0 += DFT_WARPS * DFT_EB)
#pragma unroll
        for (int j = 0; j < DFT_EB; ++j)
            if (e0 + j < nE) accs[(e0 + j) * DFT_SER + lane] = 0.f;
    for (int ch = 0; ch < nchunks; ++ch) {
        __syncthreads();                                  // previous chunk's tile no longer read
        for (int f = warp; f < L; f += DFT_WARPS)
            xs[f * DFT_SER + lane] = live ? src[(size_t)ch * chunk_stride + (size_t)f * frame_stride] : make_float2(0.f, 0.f);
        __syncthreads();
        // a warp owns the energy groups e0 = (warp + DFT_WARPS g) DFT_EB: only it touches their sums, no barrier in this loop
        for (int e0 = warp * DFT_EB; e0 < nE; e0 += DFT_WARPS * DFT_EB) {
            float2 s[DFT_EB];
#pragma unroll
            for (int j = 0; j < DFT_EB; ++j) s[j] = make_float2(0.f, 0.f);
            for (int f = 0; f < L; ++f) {
                const float2 x = xs[f * DFT_SER + lane];
#pragma unroll
                for (int j = 0; j < DFT_EB; ++j) {
                    const int e = min(e0 + j, nE - 1);
                    const float2 w = __ldg(W + (size_t)e * L + f);
                    s[j].x = fmaf(w.x, x.x, fmaf(-w.y, x.y, s[j].x));
                    s[j].y = fmaf(w.x, x.y, fmaf(w.y, x.x, s[j].y));
                }
            }
#pragma unroll
            for (int j = 0; j < DFT_EB; ++j)
                if (e0 + j < nE) accs[(e0 + j) * DFT_SER + lane] += s[j].x * s[j].x + s[j].y * s[j].y;
        }
    }
    if (!live) return;
    float* dst = I + (size_t)p * nE * (size_t)nroi + r;
    // (each warp reads back only the sums it wrote)
    for (int e0 = warp * DFT_EB; e0 < nE; e0 += DFT_WARPS * DFT_EB)
#pragma unroll
        for (int j = 0; j < DFT_EB; ++j)
            if (e0 + j < nE) dst[(size_t)(e0 + j) * nroi] = bose[e0 + j] * accs[(e0 + j) * DFT_SER + lane];
}

int launch_spectrum_dft(tacaw_ctx* ctx, const float2* d_buf, int nprobes, int64_t nroi, int L, size_t probe_stride, size_t frame_stride,
                        int nchunks, size_t chunk_stride, const float2* d_W, const float* d_bose, int nE, float* d_I, cudaStream_t st) {
    const size_t smem = sizeof(float2) * (size_t)L * DFT_SER + sizeof(float) * (size_t)nE * DFT_SER;
    TACAW_CUDA(ctx, cudaFuncSetAttribute(k_spectrum_dft, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int64_t gx = (nroi + DFT_SER - 1) / DFT_SER;
    for (int p0 = 0; p0 < nprobes; p0 += 32768) {
        const int np = nprobes - p0 < 32768 ? nprobes - p0 : 32768;
        k_spectrum_dft<<<dim3((unsigned)gx, np), DFT_SER * DFT_WARPS, smem, st>>>(d_buf + (size_t)p0 * probe_stride, (long long)nroi, probe_stride,
                                                                                frame_stride, nchunks, chunk_stride, L, d_W, d_bose, nE,
                                                                                d_I + (size_t)p0 * nE * (size_t)nroi);
        ctx->launches++;
    }
    TACAW_CUDA(ctx, cudaGetLastError());
    return TACAW_OK;
}

// DetectorSet reduction: out[d][e][p] = sum_r w[d][r] I[p][e][r].  One warp per (p, e) row of I: float4 loads of the
// row and of up to 8 weight rows (the weights stay in L2/L1), fp32 partial sums per lane, butterfly reduction.  I is
// read once for all detectors of the call.
template <int ND>
__global__ void __launch_bounds__(256) k_detect(const float* __restrict__ I, long long nrows, long long nroi, int nE, int nprobes,
                                                const float* __restrict__ w, float* __restrict__ out) {
    const long long row = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;     // p*nE + e
    const int lane = threadIdx.x & 31;
    if (row >= nrows) return;
    const float* src = I + row * nroi;
    float acc[ND];
#pragma unroll
    for (int d = 0; d < ND; ++d) acc[d] = 0.f;
    // rows start at arbitrary alignment (nroi need not be a multiple of 4): scalar accesses, coalesced across the warp
    for (long long r = lane; r < nroi; r += 32) {
        const float v = src[r];
#pragma unroll
        for (int d = 0; d < ND; ++d) acc[d] = fmaf(__ldg(w + d * nroi + r), v, acc[d]);
    }
#pragma unroll
    for (int d = 0; d < ND; ++d) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc[d] += __shfl_xor_sync(0xffffffffu, acc[d], o);
    }
    if (lane == 0) {
        const long long p = row / nE, e = row - p * nE;
#pragma unroll
        for (int d = 0; d < ND; ++d) out[((long long)d * nE + e) * nprobes + p] = acc[d];
    }
}

int launch_detect(tacaw_ctx* ctx, const float* d_I, int nprobes, int nE, int64_t nroi, const float* d_w, int ndet, float* d_out,
                  cudaStream_t st) {
    const long long nrows = (long long)nprobes * nE;
    if (nrows == 0) return TACAW_OK;
    const unsigned blocks = (unsigned)((nrows * 32 + 255) / 256);
#define TACAW_DET_CASE(K) case K: k_detect<K><<<blocks, 256, 0, st>>>(d_I, nrows, (long long)nroi, nE, nprobes, d_w, d_out); break;
    switch (ndet) {
        TACAW_DET_CASE(1) TACAW_DET_CASE(2) TACAW_DET_CASE(3) TACAW_DET_CASE(4)
        TACAW_DET_CASE(5) TACAW_DET_CASE(6) TACAW_DET_CASE(7) TACAW_DET_CASE(8)
        default: return fail(ctx, TACAW_E_UNSUPPORTED, "tacaw_detect: 1 to 8 detectors per call");
    }
#undef TACAW_DET_CASE
    ctx->launches++;
    TACAW_CUDA(ctx, cudaGetLastError());
    return TACAW_OK;
}

int launch_spectrum(tacaw_ctx* ctx, const float2* d_buf, int nprobes, int64_t nroi, int nframes, size_t probe_stride,
                    size_t frame_stride, int nchunks, size_t chunk_stride, const float2* d_roots,
                    const float* d_window, const float* d_bose, int e_lo, int nE, float* d_I, cudaStream_t st) {
    static const bool two_exchange = [] { const char* e = getenv("TACAW_SPEC_TWO_EXCHANGE"); return e && atoi(e) != 0; }();
    if (two_exchange) {       // comparison switch: the ping-pong plan for the long series too
        switch (nframes) {
            case 512: return launch_spec_n<512>(ctx, d_buf, nprobes, nroi, probe_stride, frame_stride, nchunks, chunk_stride, d_roots, d_window, d_bose, e_lo, nE, d_I, st);
            case 1024: return launch_spec_n<1024>(ctx, d_buf, nprobes, nroi, probe_stride, frame_stride, nchunks, chunk_stride, d_roots, d_window, d_bose, e_lo, nE, d_I, st);
            case 2048: return launch_spec_n<2048>(ctx, d_buf, nprobes, nroi, probe_stride, frame_stride, nchunks, chunk_stride, d_roots, d_window, d_bose, e_lo, nE, d_I, st);
        }
    }
    switch (nframes) {
        case 8: return launch_spec_n<8>(ctx, d_buf, nprobes, nroi, probe_stride, frame_stride, nchunks, chunk_stride, d_roots, d_window, d_bose, e_lo, nE, d_I, st);
        case 16: return launch_spec_n<16>(ctx, d_buf, nprobes, nroi, probe_stride, frame_stride, nchunks, chunk_stride, d_roots, d_window, d_bose, e_lo, nE, d_I, st);
        case 32: return launch_spec_n<32>(ctx, d_buf, nprobes, nroi, probe_stride, frame_stride, nchunks, chunk_stride, d_roots, d_window, d_bose, e_lo, nE, d_I, st);
        case 64: return launch_spec_n<64>(ctx, d_buf, nprobes, nroi, probe_stride, frame_stride, nchunks, chunk_stride, d_roots, d_window, d_bose, e_lo, nE, d_I, st);
        case 128: return launch_spec_n<128>(ctx, d_buf, nprobes, nroi, probe_stride, frame_stride, nchunks, chunk_stride, d_roots, d_window, d_bose, e_lo, nE, d_I, st);
        case 256: return launch_spec_n<256>(ctx, d_buf, nprobes, nroi, probe_stride, frame_stride, nchunks, chunk_stride, d_roots, d_window, d_bose, e_lo, nE, d_I, st);
        case 512: return launch_spec2_n<512>(ctx, d_buf, nprobes, nroi, probe_stride, frame_stride, nchunks, chunk_stride, d_roots, d_window, d_bose, e_lo, nE, d_I, st);
        case 1024: return launch_spec2_n<1024>(ctx, d_buf, nprobes, nroi, probe_stride, frame_stride, nchunks, chunk_stride, d_roots, d_window, d_bose, e_lo, nE, d_I, st);
        case 2048: return launch_spec2_n<2048>(ctx, d_buf, nprobes, nroi, probe_stride, frame_stride, nchunks, chunk_stride, d_roots, d_window, d_bose, e_lo, nE, d_I, st);
    }
    return fail(ctx, TACAW_E_UNSUPPORTED, "nframes must be a power of two in [8, 2048]");
}

}  // namespace tacaw

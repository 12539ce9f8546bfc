// generic.cu -- slice-step kernels for grids that are NOT powers of two: even N = 2^a 3^b 5^c 7^d <= 2048, e.g. the paper's
// 1680 = 2^4 * 3 * 5 * 7 ("1680 x 1680").
//
// Same operations, modes, layouts and normalisation as k_row / k_col of propagate.cu (O4-O7): the row kernel
// does  IFFT_x -> x t_n -> FFT_x  on the in-band columns of the mixed (kx, y) layout, the column kernel  FFT_y -> x Px Py M ->
// IFFT_y  on tiles of adjacent in-band columns.  What differs is the transform: a mixed-radix Stockham autosort FFT in
// shared memory (radices 8, 7, 6, 5, 4, 3, 2 chosen greedily on the host; each pass = N/R radix-R butterflies written as
// R-term sums over a table of the N-th roots of unity), one CTA per row / per column tile, ping-pong buffers.  It is the
// plain formulation, about 4x the arithmetic of the register FFTs of fft2.cuh and without their prefetching: a correct
// path for the paper's grid, not a tuned one.
#include "ctx.h"

namespace tacaw {

namespace {

constexpr int GEN_MAX_PASSES = 12;
constexpr int GEN_THREADS = 256;

struct GenPlan {
    int n, npass;
    int radix[GEN_MAX_PASSES];
};

bool make_plan(int n, GenPlan* pl) {
    pl->n = n;
    pl->npass = 0;
    static const int cand[7] = {8, 7, 6, 5, 4, 3, 2};
    for (int r : cand)
        while (n % r == 0) {
            if (pl->npass == GEN_MAX_PASSES) return false;
            pl->radix[pl->npass++] = r;
            n /= r;
        }
    return n == 1;
}

__device__ __forceinline__ float2 cmulg(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ float2 cfmag(float2 a, float2 b, float2 c) {
    return make_float2(fmaf(a.x, b.x, fmaf(-a.y, b.y, c.x)), fmaf(a.x, b.y, fmaf(a.y, b.x, c.y)));
}

// One Stockham pass over WC interleaved sequences of length N held as in[i * WC + c]:
//   butterfly j (0 <= j < N/R), k = j mod Ns:  v_r = in[j + r N/R] w_{Ns R}^{k r};  out[(j - k) R + k + s Ns] = sum_r v_r w_R^{s r}
// with w_M = exp(-+2 pi i / M) taken from the table roots[m] = exp(-2 pi i m / N) (conjugated for the inverse).
template <int R, bool INV>
__device__ __forceinline__ void gen_pass(const float2* __restrict__ in, float2* __restrict__ out, const float2* __restrict__ roots,
                                         int N, int Ns, int WC, int lt) {
    const int NR = N / R;
    float2 wR[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        wR[r] = roots[r * NR];
        if (INV) wR[r].y = -wR[r].y;
    }
    const int tmul = N / (Ns * R);
    for (int q = lt; q < NR * WC; q += GEN_THREADS) {
        const int j = q / WC, c = q - j * WC;
        const int k = j % Ns;
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            float2 x = in[(j + r * NR) * WC + c];
            if (r > 0) {
                float2 w = roots[k * tmul * r];
                if (INV) w.y = -w.y;
                x = cmulg(x, w);
            }
            v[r] = x;
        }
        const int j0 = (j - k) * R + k;
#pragma unroll
        for (int s = 0; s < R; ++s) {
            float2 acc = v[0];
#pragma unroll
            for (int r = 1; r < R; ++r) acc = cfmag(v[r], wR[(s * r) % R], acc);
            out[(j0 + s * Ns) * WC + c] = acc;
        }
    }
}

// All passes; the caller has made `a` visible to the CTA (barrier).  Returns the buffer that holds the result (natural order),
// visible to every thread.
template <bool INV>
__device__ float2* gen_fft(float2* a, float2* b, const float2* roots, const GenPlan& pl, int WC, int lt) {
    int Ns = 1;
    for (int i = 0; i < pl.npass; ++i) {
        const int R = pl.radix[i];
        switch (R) {
            case 2: gen_pass<2, INV>(a, b, roots, pl.n, Ns, WC, lt); break;
            case 3: gen_pass<3, INV>(a, b, roots, pl.n, Ns, WC, lt); break;
            case 4: gen_pass<4, INV>(a, b, roots, pl.n, Ns, WC, lt); break;
            case 5: gen_pass<5, INV>(a, b, roots, pl.n, Ns, WC, lt); break;
            case 6: gen_pass<6, INV>(a, b, roots, pl.n, Ns, WC, lt); break;
            case 7: gen_pass<7, INV>(a, b, roots, pl.n, Ns, WC, lt); break;
            default: gen_pass<8, INV>(a, b, roots, pl.n, Ns, WC, lt); break;
        }
        __syncthreads();
        Ns *= R;
        float2* t = a;
        a = b;
        b = t;
    }
    return a;
}

// ------------------------------------------------------------------------------------------ row kernel
// One CTA per (row y, wave): the modes of k_row (ctx.h RowMode).  Shared memory: roots [N] | A [N] | B [N].
template <int MODE>
__global__ void __launch_bounds__(GEN_THREADS) k_row_gen(RowArgs a, GenPlan pl) {
    constexpr bool HAS_T = (MODE == ROW_FIRST || MODE == ROW_MID);
    extern __shared__ __align__(16) float2 gsm[];
    const int N = pl.n, lt = threadIdx.x;
    float2* roots = gsm;
    float2* A = gsm + N;
    float2* B = A + N;
    const long long item = blockIdx.x;
    const int y = (int)(item / a.ntuples), p = (int)(item - (long long)y * a.ntuples);
    const int wv = a.tuples ? a.tuples[p] : p;
    const size_t npix = (size_t)a.ny * N;
    for (int i = lt; i < N; i += GEN_THREADS) roots[i] = a.roots[i];
    float2* row = a.waves + (size_t)wv * npix + (size_t)y * N;
    if constexpr (MODE == ROW_FIRST) {
        const float2* src = (a.probes ? a.probes + (size_t)a.wave_probe[wv] * npix : a.waves + (size_t)wv * npix) + (size_t)y * N;
        for (int i = lt; i < N; i += GEN_THREADS) A[i] = src[i];
    } else {
        for (int i = lt; i < N; i += GEN_THREADS) A[i] = (i <= a.hmax || i >= N - a.hmax) ? row[i] : make_float2(0.f, 0.f);
    }
    __syncthreads();
    float2* cur = A;
    float2* oth = B;
    if constexpr (MODE != ROW_FIRST) {
        cur = gen_fft<true>(A, B, roots, pl, 1, lt);
        oth = (cur == A) ? B : A;
    }
    if constexpr (HAS_T) {
        const int f = a.wave_frame[wv];
        const float2* tp = a.trans[(size_t)f * a.nseg + a.seg] + (size_t)a.slice * npix + (size_t)y * N;
        for (int i = lt; i < N; i += GEN_THREADS) cur[i] = cmulg(cur[i], tp[i]);
        __syncthreads();
        cur = gen_fft<false>(cur, oth, roots, pl, 1, lt);
        for (int i = lt; i < N; i += GEN_THREADS)
            if (i <= a.hmax || i >= N - a.hmax) row[i] = cur[i];
    } else if constexpr (MODE == ROW_LAST) {
        for (int i = lt; i < N; i += GEN_THREADS) row[i] = cur[i];
    } else {      // ROW_TRANS: t = exp(i sigma v), v = Re(x)/(lx ly)
        for (int i = lt; i < N; i += GEN_THREADS) {
            float s, c;
            sincosf(a.scale * cur[i].x, &s, &c);
            row[i] = make_float2(c, s);
        }
    }
}

// ------------------------------------------------------------------------------------------ column kernel
// One CTA per (group of WC adjacent columns, wave): the modes of k_col (ctx.h ColMode).  Shared memory:
// roots [N] | A [N][WC] | B [N][WC].  Column groups are selected like in k_col: the in-band ones (ix <= hmax or ix >= nx - hmax).
template <int MODE>
__global__ void __launch_bounds__(GEN_THREADS) k_col_gen(ColArgs a, GenPlan pl, int WC, int nlo, int nhi, int all) {
    extern __shared__ __align__(16) float2 gsm[];
    const int N = pl.n, lt = threadIdx.x;
    float2* roots = gsm;
    float2* A = gsm + N;
    float2* B = A + (size_t)N * WC;
    const long long item = blockIdx.x;
    const int gi = (int)(item / a.nwaves), w = (int)(item - (long long)gi * a.nwaves);
    const int NG = a.nx / WC;
    const int grp = (all || gi < nlo) ? gi : NG - (nlo + nhi - gi);
    const size_t npix = (size_t)N * a.nx;
    float2* wave = a.waves + (size_t)w * npix;
    for (int i = lt; i < N; i += GEN_THREADS) roots[i] = a.roots[i];
    // |k| <= kmax[ix] for row iy (k = signed index of iy)
    auto kept = [&](int iy, int km) { const int k = iy < N / 2 ? iy : N - iy; return k <= km; };      // |iy - N| = N - iy
    for (int q = lt; q < N * WC; q += GEN_THREADS) {
        const int iy = q / WC, c = q - iy * WC;
        const int ix = grp * WC + c;
        const int km = a.kmax[ix];
        // a column entirely outside the mask is never written by the row kernel; COL_INV input holds only |k| <= kmax
        const bool use = km >= 0 && (MODE != COL_INV || kept(iy, km));
        A[q] = use ? wave[(size_t)iy * a.nx + ix] : make_float2(0.f, 0.f);
    }
    __syncthreads();
    if constexpr (MODE == COL_INV) {
        float2* cur = gen_fft<true>(A, B, roots, pl, WC, lt);
        for (int q = lt; q < N * WC; q += GEN_THREADS) {
            const int iy = q / WC, c = q - iy * WC;
            wave[(size_t)iy * a.nx + grp * WC + c] = cur[q];
        }
    } else {
        float2* cur = gen_fft<false>(A, B, roots, pl, WC, lt);
        float2* oth = (cur == A) ? B : A;
        for (int q = lt; q < N * WC; q += GEN_THREADS) {
            const int iy = q / WC, c = q - iy * WC;
            const int ix = grp * WC + c;
            const int km = a.kmax[ix];
            float2 v = make_float2(0.f, 0.f);
            if (km >= 0 && kept(iy, km)) {
                float2 px = a.px[ix];
                px = make_float2(px.x * a.pscale, px.y * a.pscale);
                v = cmulg(cur[q], cmulg(px, a.py[iy]));
            }
            cur[q] = v;
        }
        __syncthreads();
        if constexpr (MODE == COL_MID) {
            cur = gen_fft<true>(cur, oth, roots, pl, WC, lt);
            for (int q = lt; q < N * WC; q += GEN_THREADS) {
                const int iy = q / WC, c = q - iy * WC;
                wave[(size_t)iy * a.nx + grp * WC + c] = cur[q];
            }
        } else if constexpr (MODE == COL_LASTQ) {
            for (int q = lt; q < N * WC; q += GEN_THREADS) {
                const int iy = q / WC, c = q - iy * WC;
                wave[(size_t)iy * a.nx + grp * WC + c] = cur[q];
            }
        } else {  // COL_GATHER: phi of the ROI pixels of these columns straight into buf[p][f][r]
            float2* gdst = a.gbuf + (size_t)a.wave_slot[w] * (size_t)a.gq;
            for (int q = lt; q < N * WC; q += GEN_THREADS) {
                const int iy = q / WC, c = q - iy * WC;
                const int rr = a.roi_inv[(size_t)iy * a.nx + grp * WC + c];
                if (rr >= 0) gdst[rr] = cur[q];
            }
        }
    }
}

// zero columns [c0, c1) of every row of every wave (out-of-band part of the exit wave Psi_S, O7)
__global__ void k_zero_cols_gen(float2* __restrict__ waves, long long nrows, int nx, int c0, int c1) {
    const int width = c1 - c0;
    const long long total = nrows * width;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const long long r = i / width;
        waves[r * nx + c0 + (int)(i - r * width)] = make_float2(0.f, 0.f);
    }
}

template <class K>
int opt_in_smem(tacaw_ctx* ctx, K kern, size_t smem) {
    const void* key = (const void*)kern;
    auto it = ctx->kernel_occ.find(key);
    if (it == ctx->kernel_occ.end() || (size_t)it->second < smem) {
        if (smem > 48 * 1024) TACAW_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        ctx->kernel_occ[key] = (int)smem;
    }
    return TACAW_OK;
}

}  // namespace

bool generic_grid_supported(int n) {
    GenPlan pl;
    return n >= 16 && n <= 2048 && (n % 2) == 0 && make_plan(n, &pl);
}

int launch_row_generic(tacaw_ctx* ctx, int mode, const RowArgs& a0, cudaStream_t st) {
    GenPlan pl;
    const int N = ctx->grid.nx;
    if (!make_plan(N, &pl)) return fail(ctx, TACAW_E_UNSUPPORTED, "nx must be even with prime factors 2, 3, 5, 7 only");
    RowArgs a = a0;
    if (!a.tuples) a.ntuples = a.nwaves;                 // one wave per tuple on this path (row_tuple_size() == 1)
    const long long items = (long long)a.ny * a.ntuples;
    if (items <= 0) return TACAW_OK;
    const size_t smem = sizeof(float2) * 3 * (size_t)N;
    auto go = [&](auto kern) -> int {
        if (int rc = opt_in_smem(ctx, kern, smem)) return rc;
        kern<<<(unsigned)items, GEN_THREADS, smem, st>>>(a, pl);
        ctx->launches++;
        TACAW_CUDA(ctx, cudaGetLastError());
        return TACAW_OK;
    };
    switch (mode) {
        case ROW_FIRST: return go(k_row_gen<ROW_FIRST>);
        case ROW_MID: return go(k_row_gen<ROW_MID>);
        case ROW_LAST: return go(k_row_gen<ROW_LAST>);
        case ROW_TRANS: return go(k_row_gen<ROW_TRANS>);
    }
    return fail(ctx, TACAW_E_ARG, "bad row mode");
}

int launch_col_generic(tacaw_ctx* ctx, int mode, const ColArgs& a, int ny, cudaStream_t st) {
    GenPlan pl;
    if (!make_plan(ny, &pl)) return fail(ctx, TACAW_E_UNSUPPORTED, "ny must be even with prime factors 2, 3, 5, 7 only");
    const int WC = (a.nx % 4 == 0) ? 4 : 2;              // adjacent columns per CTA (nx is even)
    const int NG = a.nx / WC;
    const int nlo = a.hmax / WC + 1, nhi = (a.hmax + WC - 1) / WC;
    const int all = nlo + nhi >= NG;
    const int ngroups = all ? NG : nlo + nhi;
    const long long items = (long long)ngroups * a.nwaves;
    if (items <= 0) return TACAW_OK;
    const size_t smem = sizeof(float2) * ((size_t)ny + 2 * (size_t)ny * WC);
    auto go = [&](auto kern) -> int {
        if (int rc = opt_in_smem(ctx, kern, smem)) return rc;
        kern<<<(unsigned)items, GEN_THREADS, smem, st>>>(a, pl, WC, nlo, nhi, all);
        ctx->launches++;
        TACAW_CUDA(ctx, cudaGetLastError());
        return TACAW_OK;
    };
    int rc = TACAW_E_ARG;
    switch (mode) {
        case COL_MID: rc = go(k_col_gen<COL_MID>); break;
        case COL_LASTQ: rc = go(k_col_gen<COL_LASTQ>); break;
        case COL_INV: rc = go(k_col_gen<COL_INV>); break;
        case COL_GATHER: rc = go(k_col_gen<COL_GATHER>); break;
        default: return fail(ctx, TACAW_E_ARG, "bad column mode");
    }
    if (rc) return rc;
    if (mode == COL_LASTQ && !all) {
        const int c0 = nlo * WC, c1 = (NG - nhi) * WC;
        const long long nrows = (long long)a.nwaves * ny;
        long long blocks = (nrows * (c1 - c0) + 255) / 256;
        if (blocks > ctx->num_sms * 16) blocks = ctx->num_sms * 16;
        k_zero_cols_gen<<<(unsigned)blocks, 256, 0, st>>>(a.waves, nrows, a.nx, c0, c1);
        ctx->launches++;
        TACAW_CUDA(ctx, cudaGetLastError());
    }
    return TACAW_OK;
}

// table of the transforms of length n on this path: the n-th roots of unity exp(-2 pi i m / n), built in fp64
void generic_host_table(int n, float2* tab) {
    for (int m = 0; m < n; ++m) {
        const double ang = -2.0 * M_PI * (double)m / (double)n;
        tab[m] = make_float2((float)cos(ang), (float)sin(ang));
    }
}

}  // namespace tacaw

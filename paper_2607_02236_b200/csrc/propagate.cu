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
//
// Both kernels are built on the single-exchange transforms of fft2.cuh: ncu shows the slice step bound
// by L1TEX (shared-memory wavefronts), so each 1D transform crosses shared memory once, wave rows and
// columns go global <-> registers directly, and only what is reused (the t_n rows shared by the probes
// of a frame, the Py table, the twiddles) is kept in shared memory.
#include <cuda.h>

#include <cstdlib>

#include "ctx.h"
#include "fft2.cuh"

// 2048-point row kernel: teams (rows in flight) per CTA, and where the 8 KB combine table of the pair plan lives.
// 2 teams + table in global memory (read through L1): 74.5 KB per CTA, three CTAs = 12 warps per SM
#ifndef TACAW_ROW2048_TEAMS
#define TACAW_ROW2048_TEAMS 2
#endif
#ifndef TACAW_ROW2048_MINB
#define TACAW_ROW2048_MINB 3
#endif
#ifndef TACAW_COL2048_REGCAP
#define TACAW_COL2048_REGCAP 1
#endif
#ifndef TACAW_COL2048_MERGE
#define TACAW_COL2048_MERGE 0
#endif
#ifndef TACAW_ROW2048_CW_SMEM
#define TACAW_ROW2048_CW_SMEM 0
#endif
// combine twiddles of the row kernel computed from w^kq and compile-time constants instead of read from the table
#ifndef TACAW_ROW2048_CW_COMPUTE
#define TACAW_ROW2048_CW_COMPUTE 1
#endif

namespace tacaw {

// Which of a thread's elements x[tid + T*m] are inside the band |h| <= H (index <= H or >= N - H).
// BAND: H = N/3 exactly (square cell with the 2/3 mask) -- the structure is known at compile time:
// chunks m < M_LO and m > M_HI are inside, chunks between are outside, the two edge chunks depend on
// tid only.  Otherwise H is a run-time value and every element is tested.
template <int N, int T, bool BAND>
struct Band {
    static constexpr int H = N / 3;
    static constexpr int M_LO = H / T, M_HI = (N - H) / T;
    bool lo_ok, hi_ok;
    int h;
    __device__ __forceinline__ Band(int tid, int hrun) : lo_ok(tid <= H - T * M_LO), hi_ok(tid >= (N - H) - T * M_HI), h(hrun) {}
    // compile-time "certainly outside"
    static constexpr __host__ __device__ bool never(int m) { return BAND && m > M_LO && m < M_HI; }
    __device__ __forceinline__ bool in(int m, int tid) const {
        if constexpr (BAND) {
            return (m < M_LO) || (m > M_HI) || (m == M_LO && lo_ok) || (m == M_HI && hi_ok);
        } else {
            const int ix = tid + T * m;
            return ix <= h || ix >= N - h;
        }
    }
};

// ------------------------------------------------------------------------------------------
template <int N>
struct RowCfg {
    using X = XPlan<N>;
    static constexpr int E = X::E, T = X::T;
    static constexpr int TEAM = (T < 32) ? 32 : T;          // threads that share an exchange buffer
    static constexpr int RPT = TEAM / T;                    // rows (one per wave of a tuple) a team transforms at once
    static constexpr int TEAMS = (N >= 2048) ? TACAW_ROW2048_TEAMS : 4;       // teams per CTA
    static constexpr int THREADS = TEAMS * TEAM;
    static constexpr int XE = X::exch(1);                   // exchange elements per row
    // three CTAs (12 warps) per SM at every size: at 2048 this caps the pair-plan kernel at 168 registers (it took 174
    // with the cap at 255), TACAW_ROW2048_MINB=1 restores two CTAs (8 warps) per SM
    static constexpr int MINB = (N >= 2048) ? TACAW_ROW2048_MINB : 3;
    static constexpr bool CW_SMEM = !X::PAIR || (TACAW_ROW2048_CW_SMEM != 0);
    static constexpr int TW = CW_SMEM ? X::TW_ELEMS : X::P::TW_ELEMS;     // twiddle entries held in shared memory
    // staged t_n row: in the paired ownership a lane pair reads elements 512 apart, i.e. the same banks; every block of 512
    // elements is therefore shifted by 8 more elements (16 banks), which keeps the half-warp wavefronts conflict free
    static constexpr int TROW = X::PAIR ? N + 8 * (N / 512) : N;
    static constexpr __host__ __device__ int tskew(int i) { return X::PAIR ? i + 8 * (i >> 9) : i; }
    static constexpr size_t smem(bool has_t) {
        return sizeof(float2) * ((size_t)TW + (size_t)TEAMS * (RPT * XE + (has_t ? TROW : 0)));
    }
};

// A team transforms row y of the RPT waves of a "tuple" at once (RPT = 2 at 256^2 and 512^2: one row per
// half warp).  The waves of a tuple belong to the same frame, so they share ONE staged t_n row, read
// back as a broadcast.  Work items are (row, tuple) pairs, flattened as y*ntuples + p and dealt out in
// equal contiguous ranges to the teams of a grid that fills the machine; consecutive items of a team share
// the row, so its t_n row is reloaded only when the frame (or the row) changes.
// The rows of the NEXT item are prefetched with cp.async into the team's exchange buffer as soon as the
// last exchange of the current item has been read back (the buffer is idle during the last pass and
// the stores), so global latency overlaps arithmetic without a staging buffer of its own.
template <int N, int MODE, bool BAND>
__global__ void __launch_bounds__(RowCfg<N>::THREADS, RowCfg<N>::MINB) k_row(RowArgs a) {
    using C = RowCfg<N>;
    using X = XPlan<N>;
    constexpr int E = C::E, T = C::T, TEAM = C::TEAM, RPT = C::RPT;
    constexpr bool HAS_T = (MODE == ROW_FIRST || MODE == ROW_MID);
    constexpr bool FULL_IN = (MODE == ROW_FIRST);           // the input row is an r-space row: no band
    extern __shared__ __align__(16) float2 smem[];
    const int lt = threadIdx.x;
    const int team = lt / TEAM, l = lt % TEAM;
    const int g = l / T, tid = l % T;
    float2* tw = smem;
    float2* exw = smem + C::TW + (size_t)team * (RPT * C::XE + (HAS_T ? C::TROW : 0));   // team's exchange rows
    float2* ex = exw + (size_t)g * C::XE;
    float2* sT = exw + (size_t)RPT * C::XE;                                              // [N]
    pdl_launch_dependents();
    xplan_load_twiddles<N, C::CW_SMEM>(tw, a.roots, lt, C::THREADS);
    const XThread<N, 1, X::PAIR && (TACAW_ROW2048_CW_COMPUTE != 0)> xt(tw, C::CW_SMEM ? tw + X::P::TW_ELEMS : a.roots + X::P::TW_ELEMS, tid, 0);
    const Band<N, T, BAND> band(tid, a.hmax);

    const long long gteam = (long long)blockIdx.x * C::TEAMS + team;
    const long long i0 = gteam * a.ipc;
    const long long i1 = min(i0 + (long long)a.ipc, a.nitems);
    const size_t npix = (size_t)a.ny * N;
    int y = 0, p = 0;
    if (i0 < i1) {
        y = (int)(i0 / a.ntuples);
        p = (int)(i0 - (long long)y * a.ntuples);
    }
    // wave of member r of tuple pv (a short last tuple repeats its last wave: identical work, identical stores)
    auto member = [&](int pv, int r) {
        return a.tuples ? __ldg(a.tuples + (size_t)pv * RPT + r) : min(pv * RPT + r, a.nwaves - 1);
    };
    // 16-byte chunks (two elements) of the row of every member; chunk cch is wanted if it touches the band
    const int clo = a.hmax / 2, chi = (N - a.hmax) / 2;
    // RCONST: the member a chunk belongs to is known at compile time (k / (NCHR/TEAM)), so the member waves are
    // looked up once per item, ahead of time (wm[]); otherwise (tiny grids) each chunk looks its member up
    constexpr int NCHR = N / 2;
    constexpr bool RCONST = (NCHR % TEAM == 0);
    constexpr int NWM = RCONST ? RPT : 1;
    auto load_members = [&](int pv, int (&wm)[NWM]) {
        if constexpr (RCONST) {
#pragma unroll
            for (int r = 0; r < RPT; ++r) wm[r] = member(pv, r);
        }
    };
    auto own_member = [&](int pv, const int (&wm)[NWM]) {
        if constexpr (RCONST) {
            int wv = wm[0];
#pragma unroll
            for (int r = 1; r < RPT; ++r) wv = (g == r) ? wm[r] : wv;
            return wv;
        } else {
            return member(pv, g);
        }
    };
    auto issue_wave = [&](int pv, int yv, const int (&wm)[NWM]) {
        constexpr int K = RPT * NCHR / TEAM;
        const float2* base[NWM];
        if constexpr (RCONST) {
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                if constexpr (MODE == ROW_FIRST) base[r] = a.probes ? a.probes + (size_t)a.wave_probe[wm[r]] * npix : a.waves + (size_t)wm[r] * npix;
                else base[r] = a.waves + (size_t)wm[r] * npix;
                base[r] += (size_t)yv * N;
            }
        }
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const int id = l + TEAM * k;
            const int r = id / NCHR, cch = id % NCHR;
            bool want = true;
            if (!FULL_IN) {
                if (BAND && RCONST) {
                    // cch = l + TEAM*(k % (NCHR/TEAM)): classify the 32-chunk block at compile time
                    constexpr int CLO = (N / 3) / 2, CHI = (N - N / 3) / 2;
                    constexpr int BPR = NCHR / TEAM > 0 ? NCHR / TEAM : 1;     // 32-chunk blocks per row
                    const int lo = TEAM * (k % BPR), hi = lo + TEAM - 1;
                    if (hi <= CLO || lo >= CHI) want = true;
                    else if (lo > CLO && hi < CHI) want = false;
                    else want = (cch <= CLO || cch >= CHI);
                } else {
                    want = (cch <= clo || cch >= chi);
                }
            }
            if (want) {
                const float2* src;
                if constexpr (RCONST) {
                    constexpr int BPR = NCHR / TEAM > 0 ? NCHR / TEAM : 1;
                    src = base[k / BPR];
                } else {
                    const int wv = member(pv, r);
                    if constexpr (MODE == ROW_FIRST) src = a.probes ? a.probes + (size_t)a.wave_probe[wv] * npix : a.waves + (size_t)wv * npix;
                    else src = a.waves + (size_t)wv * npix;
                    src += (size_t)yv * N;
                }
                cp_async16(exw + r * C::XE + 2 * cch, src + 2 * cch);
            }
        }
        cp_async_commit();
    };
    const unsigned long long pol_t = l2_policy_evict_first();     // t_n is read once per group: do not keep it in L2
    auto issue_t = [&](int f, int yv) {
        const float2* tp = a.trans[(size_t)f * a.nseg + a.seg] + (size_t)a.slice * npix + (size_t)yv * N;
        constexpr int KT = (N / 2 + TEAM - 1) / TEAM;
#pragma unroll
        for (int j = 0; j < KT; ++j)
            if (N / 2 >= TEAM * KT || l + TEAM * j < N / 2) cp_async16_hint(sT + C::tskew(2 * (l + TEAM * j)), tp + 2 * (l + TEAM * j), pol_t);
        cp_async_commit();
    };

    auto body = [&](auto sync) {
        // nothing before this point reads what the previous kernel of the stream wrote
        int cur_f = -1, cur_y = -1;
        int wv = 0, f_next = 0;
        int wm[NWM] = {0};
        bool t_new = false;
        if (i0 < i1) {
            load_members(p, wm);
            wv = own_member(p, wm);
            if constexpr (HAS_T) {
                // t_n was written long before the previous kernel: stage it while that kernel drains
                cur_f = a.wave_frame[wv];
                cur_y = y;
                issue_t(cur_f, y);
                t_new = true;
            }
        }
        pdl_wait();
        if (i0 < i1) issue_wave(p, y, wm);
        if (i0 >= i1) cp_async_wait_all();                   // twiddles are the oldest group
        else if (HAS_T) cp_async_wait_group<2>();
        else cp_async_wait_group<1>();
        __syncthreads();                          // twiddle table complete (every thread of the CTA gets here)
        if (i0 >= i1) return;
        for (long long i = i0; i < i1; ++i) {
            if constexpr (HAS_T) {
                if (i > i0) {
                    const int f = f_next;
                    t_new = (f != cur_f || y != cur_y);
                    if (t_new) {
                        cur_f = f;
                        cur_y = y;
                        sync();        // every thread of the team is done with the previous t row
                        issue_t(f, y);
                    }
                }
            }
            // this item's rows were prefetched into the exchange buffer; a t row issued after them may still fly.
            // (first item: the t row is older than the rows, both are waited for here)
            if (t_new && i > i0) cp_async_wait_group<1>();
            else cp_async_wait_all();
            sync();
            float2 x[E];
#pragma unroll
            for (int m = 0; m < E; ++m) {
                if (FULL_IN) x[m] = ex[xt.mid(m)];          // r-space row, straight into the second transform
                else if (Band<N, T, BAND>::never(m)) x[m] = make_float2(0.f, 0.f);
                else x[m] = band.in(m, tid) ? ex[tid + T * m] : make_float2(0.f, 0.f);
            }
            float2* wrow = a.waves + (size_t)wv * npix + (size_t)y * N + tid;
            // next item
            int pn = p + 1, yn = y;
            if (pn == a.ntuples) { pn = 0; ++yn; }
            const bool more = (i + 1 < i1);
            int wvn = wv;
            if (more) {
                load_members(pn, wm);
                wvn = own_member(pn, wm);
                if constexpr (HAS_T) f_next = a.wave_frame[wvn];
            }
            auto post = [&]() {
                if (more) {
                    sync();        // every thread of the team has read the exchange back
                    issue_wave(pn, yn, wm);
                }
            };
            auto nopre = []() {};
            Hooks<decltype(nopre), decltype(post)> hook{nopre, post};
            NoHook nohook;
            if constexpr (MODE != ROW_FIRST) {
                if constexpr (HAS_T) xt.template first<true, true>(x, ex, sync, nohook);
                else xt.template first<true, true>(x, ex, sync, hook);
            }
            // between the transforms register m holds element xt.mid(m) of the row (== tid + T m except at 2048)
            float2* wmid = a.waves + (size_t)wv * npix + (size_t)y * N + xt.mid0;
            if constexpr (HAS_T) {
                if (t_new && i > i0) {
                    cp_async_wait_all();
                    sync();
                }
                // (mid0 < 1024 and mid_off is a multiple of 32: the skews of base and offset add up)
                const float2* st = sT + C::tskew(xt.mid0);
#pragma unroll
                for (int m = 0; m < E; ++m) x[m] = cmul(x[m], st[C::tskew(xt.mid_off(m))]);
                xt.template second<false, true>(x, ex, sync, hook);
#pragma unroll
                for (int m = 0; m < E; ++m) {
                    if (!Band<N, T, BAND>::never(m)) {
                        if (band.in(m, tid)) wrow[T * m] = x[m];
                    }
                }
            } else if constexpr (MODE == ROW_LAST) {
#pragma unroll
                for (int m = 0; m < E; ++m) wmid[xt.mid_off(m)] = x[m];
            } else {  // ROW_TRANS: t = exp(i sigma v), v = Re(x)/(lx ly)
#pragma unroll
                for (int m = 0; m < E; ++m) {
                    float s, c;
                    sincosf(a.scale * x[m].x, &s, &c);
                    wmid[xt.mid_off(m)] = make_float2(c, s);
                }
            }
            p = pn;
            y = yn;
            wv = wvn;
        }
    };
    if constexpr (TEAM == 32) body(SyncWarp{});
    else body(SyncNamed{1 + team, TEAM});
}

// Launch with programmatic dependent launch when asked: the kernel may start while its predecessor in the
// stream drains; everything it does before pdl_wait() must not depend on that predecessor.
template <class K, class... A>
static cudaError_t launch_pdl(K kern, unsigned grid, int threads, size_t smem, cudaStream_t st, bool pdl, const A&... a) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(threads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    static const bool pdl_on = [] {
        const char* e = getenv("TACAW_PDL");
        return e ? atoi(e) != 0 : true;
    }();
    cfg.numAttrs = (pdl && pdl_on) ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, a...);
}

// grid that fills the machine exactly: occupancy x SM count CTAs.  The opt-in shared-memory attribute and the occupancy
// are per device: cached on the context (one context = one device), keyed by the kernel.
template <class K>
static int machine_ctas(tacaw_ctx* ctx, K kern, int threads, size_t smem, int* out) {
    const void* key = (const void*)kern;
    auto it = ctx->kernel_occ.find(key);
    if (it == ctx->kernel_occ.end()) {
        if (smem > 48 * 1024) TACAW_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, smem) != cudaSuccess || per_sm < 1) {
            (void)cudaGetLastError();
            per_sm = 1;
        }
        it = ctx->kernel_occ.emplace(key, per_sm).first;
    }
    // TACAW_GRID_FRAC (tuning knob, default 1): launch only this fraction of the machine-filling grid, so that kernels of
    // different streams share the machine side by side instead of one after the other
    static const double frac = [] {
        const char* e = getenv("TACAW_GRID_FRAC");
        const double v = e ? atof(e) : 1.0;
        return (v > 0.0 && v <= 1.0) ? v : 1.0;
    }();
    const int n = (int)(ctx->num_sms * it->second * frac);
    *out = n < 1 ? 1 : n;
    return TACAW_OK;
}

template <int N, int MODE, bool BAND>
static int launch_row_nb(tacaw_ctx* ctx, const RowArgs& a0, cudaStream_t st) {
    using C = RowCfg<N>;
    RowArgs a = a0;
    if (!a.tuples) a.ntuples = (a.nwaves + C::RPT - 1) / C::RPT;
    const size_t smem = C::smem(MODE == ROW_FIRST || MODE == ROW_MID);
    auto kern = k_row<N, MODE, BAND>;
    a.nitems = (long long)a.ny * a.ntuples;
    int mctas = 0;
    if (int rc = machine_ctas(ctx, kern, C::THREADS, smem, &mctas)) return rc;
    long long teams = (long long)mctas * C::TEAMS;
    if (teams > a.nitems) teams = a.nitems;
    a.ipc = (int)((a.nitems + teams - 1) / teams);
    teams = (a.nitems + a.ipc - 1) / a.ipc;
    const long long ctas = (teams + C::TEAMS - 1) / C::TEAMS;
    TACAW_CUDA(ctx, launch_pdl(kern, (unsigned)ctas, C::THREADS, smem, st, a.pdl != 0, a));
    ctx->launches++;
    TACAW_CUDA(ctx, cudaGetLastError());
    return TACAW_OK;
}

template <int N, int MODE>
static int launch_row_n(tacaw_ctx* ctx, const RowArgs& a, cudaStream_t st) {
    // ROW_FIRST reads a full r-space row; its stores use the band like the others
    if (a.hmax == N / 3) return launch_row_nb<N, MODE, true>(ctx, a, st);
    return launch_row_nb<N, MODE, false>(ctx, a, st);
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

int row_tuple_size(int nx) {
    const int t = nx / fft2_elems(nx);
    return t < 32 ? 32 / t : 1;
}

int slice_step_table_elems(int n) { return xplan_table_elems(n); }
void slice_step_host_table(int n, float2* tab) { xplan_host_table(n, tab); }

int launch_row(tacaw_ctx* ctx, int mode, const RowArgs& a, cudaStream_t st) {
    if (a.nwaves <= 0) return TACAW_OK;
    if (ctx->generic_path) return launch_row_generic(ctx, mode, a, st);      // a grid edge that is not a power of two
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
    return fail(ctx, TACAW_E_UNSUPPORTED, "nx must be a power of two in [16, 2048] on this path");
}

// ------------------------------------------------------------------------------------------
template <int N, int MODE = COL_MID>
struct ColCfg {
    using X = XPlan<N>;
    static constexpr int E = X::E, T = X::T;
    // adjacent columns transformed together.  The slice step reads its tiles from L2, where 64-byte row segments are
    // full speed; the potential pass (COL_INV at 256^2 and below) streams from HBM, where they cost a 2x over-fetch
    // (ncu: 7.4 GB read for 3.7 GB of tiles), so it takes full 128-byte lines
    static constexpr int WC = (N >= 1024) ? 4 : ((MODE == COL_INV && N <= 256) ? 16 : 8);
    static constexpr bool PY_SMEM = (N <= 512);              // Py table in shared memory (else read through L1)
    static constexpr int THREADS = T * WC;
    static constexpr int XE = X::exch(WC);
    // MERGE (2048): the TMA staging tile and the exchange buffer are ONE region (a tile is in registers before the first
    // exchange is written, and the next tile is requested only after the last exchange of the item has been read back):
    // 84 KB instead of 148 KB per CTA, so two CTAs (16 warps) fit an SM
    static constexpr bool MERGE = X::PAIR && (TACAW_COL2048_MERGE != 0);
    static constexpr int MINB = (N <= 1024) ? 3 : (MERGE ? 2 : 1);
    // Register cap through the thread count of __launch_bounds__ (a launch may use fewer threads than it declares): 2048 runs
    // one 256-thread CTA per SM (shared memory), and ptxas then takes 226 registers because it may.  Declared for 384 threads
    // the cap is 168 (no spills; 400 threads already round up to 16 warps and a cap of 128, which spills), which leaves room for one row-kernel CTA of the other stream's wave group on the same SM
    // (256 x 168 + 128 x 168 registers, 149 + 75 KB of shared memory).
    static constexpr int LB_THREADS = (X::PAIR && !MERGE && TACAW_COL2048_REGCAP) ? 384 : THREADS;
    // twiddles | Py | (pad to 128 B) staging tile [N][WC] (TMA destination) | exchange | mbarrier
    static constexpr int OFF_S = ((X::TW_ELEMS + (PY_SMEM ? N : 0)) + 15) / 16 * 16;
    static constexpr int RB = (N < 256) ? N : 256;            // rows per TMA box
    static constexpr int OFF_X = OFF_S + (MERGE ? 0 : N * WC);
    static_assert(!MERGE || XE >= N * WC, "merged region must hold a tile");
    static constexpr size_t smem() { return sizeof(float2) * ((size_t)OFF_X + XE + 2); }
};

// Work items of a column launch are (column group, wave) pairs, flattened as gi*nwaves + w over the
// selected groups (the in-band ones, or all of them when hmax covers the grid) and dealt out in equal
// contiguous ranges to a machine-filling grid, like the row kernel.  The [N][WC] tile of the NEXT item is
// staged by TMA while the current one is transformed.
// BAND: every kmax[ix] <= N/3, so the chunks of k strictly between N/3 and N - N/3 are masked for
// every column and are neither multiplied nor tested (single-exchange plans; the pair plan tests every element).
template <int N, int MODE, bool BAND>
__global__ void __launch_bounds__(ColCfg<N, MODE>::LB_THREADS, ColCfg<N, MODE>::MINB) k_col(ColArgs a, const __grid_constant__ CUtensorMap tm) {
    using C = ColCfg<N, MODE>;
    using X = XPlan<N>;
    constexpr int E = C::E, T = C::T, WC = C::WC;
    constexpr bool MERGE = C::MERGE;
    extern __shared__ __align__(128) float2 smem[];
    const int lt = threadIdx.x;
    const int c = lt % WC, tid = lt / WC;
    float2* tw = smem;
    float2* sPy = smem + X::TW_ELEMS;             // Py[ky]
    float2* sS = smem + C::OFF_S;                 // staging tile
    float2* ex = smem + C::OFF_X;                 // exchange buffer (the same region when MERGE)
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(ex + C::XE);
    pdl_launch_dependents();
    if (lt == 0) {
        mbar_init(bar, 1);
        mbar_init_fence();
    }
    xplan_load_twiddles<N>(tw, a.roots, lt, C::THREADS);
    if constexpr (MODE != COL_INV && C::PY_SMEM) {
        for (int i = lt; i < N / 2; i += C::THREADS) cp_async16(sPy + 2 * i, a.py + 2 * i);
        cp_async_commit();
    }
    const XThread<N, WC> xt(tw, tw + X::P::TW_ELEMS, tid, c);
    const int NG = a.nx / WC;
    const int nlo = a.hmax / WC + 1;            // groups covering ix in [0, hmax]
    const int nhi = (a.hmax + WC - 1) / WC;     // groups covering ix in [nx-hmax, nx)
    const bool all = (nlo + nhi >= NG);
    auto group_of = [&](int gi) { return (all || gi < nlo) ? gi : NG - (nlo + nhi - gi); };
    const long long i0 = (long long)blockIdx.x * a.ipc;
    const long long i1 = min(i0 + (long long)a.ipc, a.nitems);
    const size_t npix = (size_t)N * a.nx;
    using B = Band<N, T, BAND && !X::PAIR>;
    // tile of wave wv, column group grp -> staging: one TMA box of [RB rows][WC columns] per RB rows, issued by one
    // thread, completion counted in bytes on the mbarrier (every thread has passed a barrier after its last read of sS)
    auto issue_tile = [&](int wv, int grp) {
        if (lt == 0) {
            fence_proxy_async();
            mbar_expect_tx(bar, (unsigned)(N * WC * sizeof(float2)));
#pragma unroll
            for (int b = 0; b < N / C::RB; ++b) tma_load_2d(sS + b * C::RB * WC, &tm, grp * WC, (a.wave0 + wv) * N + b * C::RB, bar);
        }
    };
    unsigned parity = 0;

    auto body = [&](auto sync) {
        int gi = 0, w = 0;
        pdl_wait();                              // the tables above do not depend on the previous kernel; the waves do
        if (i0 < i1) {
            gi = (int)(i0 / a.nwaves);
            w = (int)(i0 - (long long)gi * a.nwaves);
            issue_tile(w, group_of(gi));
        }
        cp_async_wait_all();
        sync();                                  // tables and the first tile visible
        if (i0 >= i1) return;
        int cur_gi = -1;
        float2 px = make_float2(0.f, 0.f);
        int km = -1;
        int dlo = -1, dhi = -1;                  // |k| <= km  <=>  T*m <= dlo (m < E/2)  or  N - T*m <= dhi (m >= E/2)
        bool live = true;
        size_t coloff = 0, midoff = 0;
        for (long long i = i0; i < i1; ++i) {
            if (gi != cur_gi) {
                cur_gi = gi;
                const int ix = group_of(gi) * WC + c;
                coloff = (size_t)ix + (size_t)tid * a.nx;
                midoff = (size_t)ix + (size_t)xt.mid0 * a.nx;
                // a column entirely outside the mask is never written by the row kernel: it is not
                // used (NaN * 0 would not be 0) and comes out as zeros
                km = a.kmax[ix];
                live = km >= 0;
                dlo = km - tid;
                dhi = km + tid;
                if constexpr (MODE != COL_INV) {
                    px = a.px[ix];
                    px = make_float2(px.x * a.pscale, px.y * a.pscale);
                }
            }
            // |k| <= km for the element register m holds BETWEEN the transforms (row xt.mid(m) of the column)
            auto keep_mid = [&](int m) {
                if constexpr (X::PAIR) {
                    const int r = xt.mid0 + pair_off(m & 15);            // row in the lower half
                    return (m < 16) ? (r <= km) : (N / 2 - r <= km);      // row r + N/2 is k = r - N/2
                } else {
                    return (T * m < N / 2) ? (T * m <= dlo) : (N - T * m <= dhi);
                }
            };
            float2* wc = a.waves + (size_t)w * npix + coloff;
            float2* wmid = a.waves + (size_t)w * npix + midoff;
            const size_t rs = (size_t)T * a.nx;
            mbar_wait(bar, parity);              // this item's tile has landed
            parity ^= 1;
            float2 x[E];
#pragma unroll
            for (int m = 0; m < E; ++m) {
                // COL_INV input (V(q) or the probe aperture): only |k| <= kmax[ix] was written
                const bool keep = (MODE != COL_INV) || ((T * m < N / 2) ? (T * m <= dlo) : (N - T * m <= dhi));
                x[m] = (live && keep) ? sS[(tid + T * m) * WC + c] : make_float2(0.f, 0.f);
            }
            int wn = w + 1, gn = gi;
            if (wn == a.nwaves) { wn = 0; ++gn; }
            const bool more = (i + 1 < i1);
            sync();                              // staging tile consumed; previous exchange read back
            if constexpr (!MERGE) {
                if (more) issue_tile(wn, group_of(gn));
            }
            // MERGE: the next tile goes into the exchange region, as soon as the item's last exchange has been read back
            auto nopre = []() {};
            auto post = [&]() {
                if constexpr (MERGE) {
                    if (more) {
                        sync();
                        issue_tile(wn, group_of(gn));
                    }
                }
            };
            Hooks<decltype(nopre), decltype(post)> hook{nopre, post};
            NoHook nohook;
            if constexpr (MODE == COL_INV) {
                xt.template first<true, false>(x, ex, sync, hook);
#pragma unroll
                for (int m = 0; m < E; ++m) wmid[(size_t)xt.mid_off(m) * a.nx] = x[m];
            } else {
                if constexpr (MODE == COL_LASTQ || MODE == COL_GATHER) xt.template first<false, false>(x, ex, sync, hook);
                else xt.template first<false, false>(x, ex, sync, nohook);
#pragma unroll
                for (int m = 0; m < E; ++m) {
                    if (B::never(m)) {
                        x[m] = make_float2(0.f, 0.f);
                    } else {
                        const float2 p = cmul(px, C::PY_SMEM ? sPy[xt.mid(m)] : __ldg(a.py + xt.mid(m)));
                        x[m] = keep_mid(m) ? cmul(x[m], p) : make_float2(0.f, 0.f);
                    }
                }
                if constexpr (MODE == COL_MID) {
                    xt.template second<true, true>(x, ex, sync, hook);
#pragma unroll
                    for (int m = 0; m < E; ++m) wc[m * rs] = x[m];
                } else if constexpr (MODE == COL_GATHER) {
                    // fused a6: phi = Psi_S / sqrt(nx ny) of the ROI pixels of this column, straight into buf[p][f][r]
                    const int ixg = group_of(gi) * WC + c;
                    const int* invc = a.roi_inv + ixg + (size_t)xt.mid0 * a.nx;
                    float2* gdst = a.gbuf + (size_t)a.wave_slot[w] * (size_t)a.gq;
#pragma unroll
                    for (int m = 0; m < E; ++m) {
                        const int rr = invc[(size_t)xt.mid_off(m) * a.nx];
                        if (rr >= 0) gdst[rr] = x[m];
                    }
                } else {
#pragma unroll
                    for (int m = 0; m < E; ++m) wmid[(size_t)xt.mid_off(m) * a.nx] = x[m];
                }
            }
            w = wn;
            gi = gn;
        }
    };
    if constexpr (C::THREADS <= 32) body(SyncWarp{});
    else body(SyncBlock{});
}

// Tensor map of a stack of waves seen as a 2D array of 8-byte elements [rows][nx]; box = [box_rows][box_cols].
static int make_tile_map(tacaw_ctx* ctx, CUtensorMap* tm, const void* base, int nx, long long rows, int box_cols, int box_rows) {
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn encode = [] {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) {
            (void)cudaGetLastError();
            f = nullptr;
        }
        return (encode_fn)f;
    }();
    if (!encode) return fail(ctx, TACAW_E_CUDA, "cuTensorMapEncodeTiled is not available");
    const cuuint64_t dims[2] = {(cuuint64_t)nx, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)nx * sizeof(float2)};
    const cuuint32_t box[2] = {(cuuint32_t)box_cols, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = encode(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void*>(base), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(ctx, TACAW_E_CUDA, "cuTensorMapEncodeTiled failed (" + std::to_string((int)r) + ")");
    return TACAW_OK;
}

// Tensor maps are encoded once per wave stack and kept on the context (cuTensorMapEncodeTiled per launch costs host time on
// a path that issues one launch every few microseconds); a small FIFO, cleared when the workspace changes.
static int tile_map(tacaw_ctx* ctx, const CUtensorMap** out, const void* base, int nx, long long rows, int box_cols, int box_rows) {
    for (auto& e : ctx->maps)
        if (e.base == base && e.rows == rows && e.nx == nx && e.box_cols == box_cols && e.box_rows == box_rows) { *out = &e.tm; return TACAW_OK; }
    if (ctx->maps.size() >= 16) ctx->maps.erase(ctx->maps.begin());
    ctx->maps.emplace_back();
    auto& e = ctx->maps.back();
    e.base = base; e.rows = rows; e.nx = nx; e.box_cols = box_cols; e.box_rows = box_rows;
    int rc = make_tile_map(ctx, &e.tm, base, nx, rows, box_cols, box_rows);
    if (rc) { ctx->maps.pop_back(); return rc; }
    *out = &e.tm;
    return TACAW_OK;
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

template <int N, int MODE, bool BAND>
static int launch_col_nb(tacaw_ctx* ctx, const ColArgs& a0, cudaStream_t st) {
    using C = ColCfg<N, MODE>;
    ColArgs a = a0;
    const int NG = a.nx / C::WC;
    const int nlo = a.hmax / C::WC + 1, nhi = (a.hmax + C::WC - 1) / C::WC;
    const bool all = nlo + nhi >= NG;
    const int ngroups = all ? NG : nlo + nhi;
    const size_t smem = C::smem();
    auto kern = k_col<N, MODE, BAND>;
    a.nitems = (long long)ngroups * a.nwaves;
    int mctas = 0;
    if (int rc = machine_ctas(ctx, kern, C::THREADS, smem, &mctas)) return rc;
    long long ctas = mctas;
    if (ctas > a.nitems) ctas = a.nitems;
    a.ipc = (int)((a.nitems + ctas - 1) / ctas);
    ctas = (a.nitems + a.ipc - 1) / a.ipc;
    // one tensor map per wave stack (not per launch): the launch addresses its waves by their index in the stack
    if (!a.stack) { a.stack = a.waves; a.stack_waves = a.nwaves; a.wave0 = 0; }
    const CUtensorMap* tmp = nullptr;
    if (int rc = tile_map(ctx, &tmp, a.stack, a.nx, (long long)a.stack_waves * N, C::WC, C::RB)) return rc;
    TACAW_CUDA(ctx, launch_pdl(kern, (unsigned)ctas, C::THREADS, smem, st, a.pdl != 0, a, *tmp));
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
    // COL_INV applies no mask; the masked modes may skip the k chunks no column keeps
    const bool band = a.kmaxmax >= 0 && a.kmaxmax <= N / 3;
    switch (mode) {
        case COL_MID: return band ? launch_col_nb<N, COL_MID, true>(ctx, a, st) : launch_col_nb<N, COL_MID, false>(ctx, a, st);
        case COL_LASTQ: return band ? launch_col_nb<N, COL_LASTQ, true>(ctx, a, st) : launch_col_nb<N, COL_LASTQ, false>(ctx, a, st);
        case COL_INV: return launch_col_nb<N, COL_INV, false>(ctx, a, st);
        case COL_GATHER: return band ? launch_col_nb<N, COL_GATHER, true>(ctx, a, st) : launch_col_nb<N, COL_GATHER, false>(ctx, a, st);
    }
    return fail(ctx, TACAW_E_ARG, "bad column mode");
}

int launch_col(tacaw_ctx* ctx, int mode, const ColArgs& a, int ny, cudaStream_t st) {
    if (a.nwaves <= 0) return TACAW_OK;
    if (ctx->generic_path) return launch_col_generic(ctx, mode, a, ny, st);
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
    return fail(ctx, TACAW_E_UNSUPPORTED, "ny must be a power of two in [16, 2048] on this path");
}

}  // namespace tacaw

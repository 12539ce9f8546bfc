// potential.cu -- slice binning (a1), structure-factor potential (K1), probe fill (K3), ROI gather (K5).
//
// K1 (O2):  V_n[h,k] = sum_s f_s(q^2) sum_{j in (n,s)} exp(-2 pi i (h x_j/lx + k y_j/ly)),
// f_s(q^2) = sum_{i<4} a_si exp(-b_si q^2), on in-band (h,k) only.  The phase factorises per atom,
// exp(-2 pi i h u_j) exp(-2 pi i k v_j), so a slice is a rank-K outer-product sum; each CTA owns a
// 32 x 32 tile of the quadrant h >= 0, k >= 0, stages the per-atom phase vectors of a chunk of atoms
// in shared memory and accumulates 2x4 points per thread in registers.  v_n is real, so the other
// three quadrants follow from the same four real sums (see k_potential).
// Phases use fixed-point fractional coordinates U = round(u 2^32): (h*U mod 2^32) is exact
// integer arithmetic, then sincospif -- fp32 h*x/L would lose ~4e-4 rad at |h| ~ 1000.
#include <algorithm>
#include <cstdlib>
#include <mutex>

#include "ctx.h"

namespace tacaw {

// ---------------------------------------------------------------------------------------- a1
// key_j = (frame*nslices + slice)*nspecies + species;  fixed-point fractional coordinates.
__global__ void k_atom_keys(const double* __restrict__ pos, const int32_t* __restrict__ species, int natoms,
                            long long ntotal, int nspecies, double dz, int nslices, double z0, double inv_lx,
                            double inv_ly, int* __restrict__ keys, uint32_t* __restrict__ ux, uint32_t* __restrict__ uy,
                            int* __restrict__ counts, int* __restrict__ nclamped, int* __restrict__ flags) {
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ntotal) return;
    const int f = (int)(i / natoms), j = (int)(i - (long long)f * natoms);
    double fz = floor((pos[3 * i + 2] - z0) / dz);
    int n;
    if (fz < 0.0) { n = 0; atomicAdd(nclamped, 1); }
    else if (fz > (double)(nslices - 1)) { n = nslices - 1; atomicAdd(nclamped, 1); }
    else n = (int)fz;
    int s = species[j];
    if (s < 0 || s >= nspecies) { atomicAdd(flags, 1); s = 0; }     // sticky: reported by tacaw_device_status
    int key = (f * nslices + n) * nspecies + s;
    keys[i] = key;
    atomicAdd(counts + key, 1);
    double fx = pos[3 * i] * inv_lx, fy = pos[3 * i + 1] * inv_ly;
    fx -= floor(fx);
    fy -= floor(fy);
    ux[i] = (uint32_t)(unsigned long long)llrint(fx * 4294967296.0);   // wraps 2^32 -> 0
    uy[i] = (uint32_t)(unsigned long long)llrint(fy * 4294967296.0);
}

// exclusive scan of counts[nkeys] -> offsets[nkeys+1]; one CTA.
__global__ void k_scan_counts(const int* __restrict__ counts, int nkeys, int* __restrict__ offsets) {
    __shared__ int warp_sum[32];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int base = 0; base < nkeys; base += blockDim.x) {
        int i = base + threadIdx.x;
        int v = (i < nkeys) ? counts[i] : 0;
        int incl = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += t;
        }
        if (lane == 31) warp_sum[wid] = incl;
        __syncthreads();
        if (wid == 0) {
            int ws = (lane < nw) ? warp_sum[lane] : 0;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                int t = __shfl_up_sync(0xffffffffu, ws, d);
                if (lane >= d) ws += t;
            }
            warp_sum[lane] = ws;     // inclusive over warps
        }
        __syncthreads();
        int before = (wid > 0 ? warp_sum[wid - 1] : 0) + carry;
        if (i < nkeys) offsets[i] = before + incl - v;
        __syncthreads();
        if (threadIdx.x == 0) carry += warp_sum[nw - 1];
        __syncthreads();
    }
    if (threadIdx.x == 0) offsets[nkeys] = carry;
}

// One warp per key: stable compaction (original atom order) of the atoms of that key's frame.
__global__ void k_compact(const int* __restrict__ keys, int natoms, int nkeys_per_frame, int nkeys_total,
                          const int* __restrict__ offsets, const uint32_t* __restrict__ ux,
                          const uint32_t* __restrict__ uy, uint32_t* __restrict__ sx, uint32_t* __restrict__ sy) {
    const int key = (int)(((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
    const int lane = threadIdx.x & 31;
    if (key >= nkeys_total) return;
    const int out0 = offsets[key];
    const int cnt = offsets[key + 1] - out0;
    if (cnt == 0) return;
    const int f = key / nkeys_per_frame;
    const size_t fbase = (size_t)f * natoms;
    const int* kf = keys + fbase;
    int written = 0;
    for (int base = 0; base < natoms && written < cnt; base += 128) {
        int jj[4];
        bool hit[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            jj[u] = base + 32 * u + lane;
            hit[u] = (jj[u] < natoms) && (kf[jj[u]] == key);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            unsigned bal = __ballot_sync(0xffffffffu, hit[u]);
            if (hit[u]) {
                int o = out0 + written + __popc(bal & ((1u << lane) - 1));
                sx[o] = ux[fbase + jj[u]];
                sy[o] = uy[fbase + jj[u]];
            }
            written += __popc(bal);
        }
    }
}

// ---------------------------------------------------------------------------------------- K1
// Quadrant form.  With ex = e^{-2 pi i h u} = a + ib and ey = e^{-2 pi i k v} = c + id,
//   ex ey       = (ac - bd) + i(ad + bc)   -> V(h, k)
//   ex conj(ey) = (ac + bd) + i(bc - ad)   -> V(h,-k)
// and V(-h,-k) = conj V(h,k), V(-h,k) = conj V(h,-k) because v_n is real.  So the four real sums
// (ac, bd, ad, bc) over the atoms of a slice, for h >= 0 and k >= 0 only, give all four quadrants:
// 4 FMA per atom per point for 4 points (a direct complex sum is 4 FMA per point).
constexpr int POT_T = 32;       // tile edge in h and in k
constexpr int POT_CHUNK = 64;   // atoms staged per step
constexpr int POT_THREADS = 128;

__device__ __forceinline__ float2 phase_fixed(uint32_t u, int h) {
    // exp(-2 pi i h u/2^32): (h*u mod 2^32) as a signed fraction of a half turn
    int32_t p = (int32_t)((uint32_t)h * u);
    float s, c;
    sincospif((float)p * 4.656612873077393e-10f, &s, &c);   // p / 2^31
    return make_float2(c, -s);
}

__global__ void __launch_bounds__(POT_THREADS) k_potential(const uint32_t* __restrict__ sx, const uint32_t* __restrict__ sy,
                                                            const int* __restrict__ offsets, int nspecies, const AbTable ab,
                                                            const int* __restrict__ kmax_pot, int hmax, int nx, int ny,
                                                            float inv_lx, float inv_ly, float2* __restrict__ V) {
    // phases of the staged atoms: ex[r][atom] = e^{-2 pi i (h0+r) u}, built as coarse[r/8] * fine[r%8]
    __shared__ float2 ex[POT_T][POT_CHUNK + 1];
    __shared__ float2 ey[POT_T][POT_CHUNK + 1];
    __shared__ float2 coarse[2][4][POT_CHUNK];
    __shared__ float2 fine[2][8][POT_CHUNK];
    const int n = blockIdx.z;
    const int h0 = blockIdx.x * POT_T, k0 = blockIdx.y * POT_T;
    if (h0 > hmax || kmax_pot[h0] < k0) return;        // tile entirely outside the mask
    const int lt = threadIdx.x;
    const int th = lt & 15, tk = lt >> 4;             // 16 x 8 threads, 2 (h) x 4 (k) points each
    // per point two packed accumulators: P = (ac, ad) += a (c, d) and Q = (bc, bd) += b (c, d): two FFMA2 with a
    // broadcast scalar operand instead of four FFMA (the kernel is bound by issue slots, not by the fp32 pipe)
    float2 accP[2][4], accQ[2][4], vsP[2][4], vsQ[2][4];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) vsP[i][j] = vsQ[i][j] = make_float2(0.f, 0.f);
    for (int s = 0; s < nspecies; ++s) {
        const int a0 = offsets[n * nspecies + s], a1 = offsets[n * nspecies + s + 1];
        if (a0 == a1) continue;
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) accP[i][j] = accQ[i][j] = make_float2(0.f, 0.f);
        for (int base = a0; base < a1; base += POT_CHUNK) {
            const int cnt = min(POT_CHUNK, a1 - base);
            __syncthreads();
            for (int i = lt; i < POT_CHUNK * 24; i += POT_THREADS) {
                const int at = i % POT_CHUNK, e = i / POT_CHUNK;       // e: axis*12 + table entry
                if (at < cnt) {
                    const int axis = e / 12, j = e % 12;
                    const uint32_t u = axis ? sy[base + at] : sx[base + at];
                    if (j < 4) coarse[axis][j][at] = phase_fixed(u, (axis ? k0 : h0) + 8 * j);
                    else if (j == 4) fine[axis][0][at] = make_float2(1.f, 0.f);        // exp(0)
                    else fine[axis][j - 4][at] = phase_fixed(u, j - 4);
                }
            }
            __syncthreads();
            for (int i = lt; i < POT_CHUNK * 2 * POT_T; i += POT_THREADS) {
                const int at = i % POT_CHUNK, rr = i / POT_CHUNK;
                if (at < cnt) {
                    const int axis = rr / POT_T, r = rr % POT_T;
                    const float2 cph = coarse[axis][r >> 3][at], fph = fine[axis][r & 7][at];
                    // packed complex product (FMUL2 + FFMA2)
                    const float2 ph = __ffma2_rn(make_float2(-cph.y, cph.x), make_float2(fph.y, fph.y),
                                                 __fmul2_rn(cph, make_float2(fph.x, fph.x)));
                    if (axis) ey[r][at] = ph; else ex[r][at] = ph;
                }
            }
            __syncthreads();
#pragma unroll 4
            for (int at = 0; at < cnt; ++at) {
                float2 xh[2], yk[4];
#pragma unroll
                for (int i = 0; i < 2; ++i) xh[i] = ex[th + 16 * i][at];
#pragma unroll
                for (int j = 0; j < 4; ++j) yk[j] = ey[tk + 8 * j][at];
#pragma unroll
                for (int i = 0; i < 2; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        accP[i][j] = __ffma2_rn(yk[j], make_float2(xh[i].x, xh[i].x), accP[i][j]);
                        accQ[i][j] = __ffma2_rn(yk[j], make_float2(xh[i].y, xh[i].y), accQ[i][j]);
                    }
            }
        }
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                float qx = (float)(h0 + th + 16 * i) * inv_lx, qy = (float)(k0 + tk + 8 * j) * inv_ly;
                float q2 = qx * qx + qy * qy;
                float f = 0.f;
#pragma unroll
                for (int g = 0; g < 4; ++g) f += ab.a[s][g] * expf(-ab.b[s][g] * q2);
                vsP[i][j] = __ffma2_rn(accP[i][j], make_float2(f, f), vsP[i][j]);
                vsQ[i][j] = __ffma2_rn(accQ[i][j], make_float2(f, f), vsQ[i][j]);
            }
    }
    float2* Vn = V + (size_t)n * nx * ny;
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int h = h0 + th + 16 * i, k = k0 + tk + 8 * j;
            if (h > hmax) continue;
            if (k > kmax_pot[h]) continue;
            const float ac = vsP[i][j].x, ad = vsP[i][j].y, bc = vsQ[i][j].x, bd = vsQ[i][j].y;
            const int ixm = (nx - h) % nx, iym = (ny - k) % ny;
            Vn[(size_t)k * nx + h] = make_float2(ac - bd, ad + bc);
            if (k > 0) Vn[(size_t)iym * nx + h] = make_float2(ac + bd, bc - ad);
            if (h > 0) Vn[(size_t)iym * nx + ixm] = make_float2(ac - bd, -(ad + bc));
            if (h > 0 && k > 0) Vn[(size_t)k * nx + ixm] = make_float2(ac + bd, ad - bc);
        }
}

int launch_potential(tacaw_ctx* ctx, const double* d_pos, const int32_t* d_species, int natoms, int nframes, int nspecies,
                     const AbTable& ab, double dz, int nslices, double z0, float2* d_V, int** d_nclamped_out,
                     cudaStream_t st) {
    const int nx = ctx->grid.nx, ny = ctx->grid.ny;
    const long long ntotal = (long long)natoms * nframes;
    const long long nkeys_ll = (long long)nframes * nslices * nspecies;
    if (nkeys_ll > (1LL << 30) || ntotal > (1LL << 31) - 1) return fail(ctx, TACAW_E_UNSUPPORTED, "batch too large");
    const int nkeys = (int)nkeys_ll;
    // build region layout: clamp counter (256 B) | keys[nt] ux[nt] uy[nt] sx[nt] sy[nt] counts[nkeys] offsets[nkeys+1]
    size_t nt = (size_t)(ntotal > 0 ? ntotal : 1);
    size_t need = 256 + sizeof(int) * (5 * nt + 2 * (size_t)nkeys + 2);
    void* reg = nullptr;
    int rc = region(ctx, tacaw_ctx::R_BUILD, need, &reg, "tacaw_build_slices");
    if (rc) return rc;
    int* d_nclamped = (int*)reg;
    *d_nclamped_out = d_nclamped;
    int* keys = (int*)((char*)reg + 256);
    uint32_t* ux = (uint32_t*)(keys + nt);
    uint32_t* uy = ux + nt;
    uint32_t* sx = uy + nt;
    uint32_t* sy = sx + nt;
    int* counts = (int*)(sy + nt);
    int* offsets = counts + nkeys;
    TACAW_CUDA(ctx, cudaMemsetAsync(counts, 0, sizeof(int) * (2 * (size_t)nkeys + 1), st));
    TACAW_CUDA(ctx, cudaMemsetAsync(d_nclamped, 0, sizeof(int), st));
    // d_V is not cleared: k_potential writes every in-band (h,k), and the column pass that follows reads only those
    if (ntotal == 0) TACAW_CUDA(ctx, cudaMemsetAsync(d_V, 0, sizeof(float2) * (size_t)nframes * nslices * nx * ny, st));
    if (ntotal > 0) {
        k_atom_keys<<<(unsigned)((ntotal + 255) / 256), 256, 0, st>>>(d_pos, d_species, natoms, ntotal, nspecies, dz, nslices,
                                                                     z0, 1.0 / ctx->grid.lx_A, 1.0 / ctx->grid.ly_A, keys, ux,
                                                                     uy, counts, d_nclamped, ctx->d_flags);
        ctx->launches++;
    }
    k_scan_counts<<<1, 1024, 0, st>>>(counts, nkeys, offsets);
    ctx->launches++;
    if (ntotal > 0) {
        k_compact<<<(unsigned)(((long long)nkeys * 32 + 255) / 256), 256, 0, st>>>(keys, natoms, nslices * nspecies, nkeys, offsets,
                                                                                  ux, uy, sx, sy);
        ctx->launches++;
        const int hmax = ctx->hmax_pot;
        const int total_slices = nframes * nslices;
        // K1 on the tensor cores (potential_tc.cu) unless TACAW_K1_TC=0 asks for the fp32-pipe kernel below (kept for
        // comparison and for more than four species)
        static const bool use_tc = [] { const char* e = getenv("TACAW_K1_TC"); return e ? atoi(e) != 0 : true; }();
        if (use_tc && nspecies <= potential_tc_max_species())
            return launch_potential_tc(ctx, sx, sy, offsets, nspecies, ab, total_slices, d_V, st);
        for (int z0i = 0; z0i < total_slices; z0i += 65535) {
            int nz = total_slices - z0i < 65535 ? total_slices - z0i : 65535;
            dim3 grid((hmax + 1 + POT_T - 1) / POT_T, (ctx->kmaxmax_pot + 1 + POT_T - 1) / POT_T, nz);
            k_potential<<<grid, POT_THREADS, 0, st>>>(sx, sy, offsets + (size_t)z0i * nspecies, nspecies, ab, ctx->d_kmax_pot, hmax, nx,
                                              ny, (float)(1.0 / ctx->grid.lx_A), (float)(1.0 / ctx->grid.ly_A),
                                              d_V + (size_t)z0i * nx * ny);
            ctx->launches++;
        }
    }
    TACAW_CUDA(ctx, cudaGetLastError());
    return TACAW_OK;
}

// ---------------------------------------------------------------------------------------- a1 + K1 without a workspace
// tacaw_build_slices_static (tacaw.h): the same kernels as launch_potential, with the build region (clamp counter, keys,
// fixed-point coordinates, sorted coordinates, counts, offsets) in this file-scope device array instead of the caller's
// workspace, for callers that cannot allocate.  Every GPU that loads the library holds the array until the process exits.
// All calls on a device share it and it keeps the previous call's contents: the counters are cleared on the caller's
// stream at the start of every call, and two calls that overlap on the GPU race.
static __device__ __align__(256) unsigned char g_static_build[TACAW_STATIC_SCRATCH_BYTES];

// In host code `g_static_build` is only a handle for the runtime, not a device address: resolve it once per device, with
// that device current (TACAW_ENTER in the entry point), and hand the kernels the resolved pointer.
constexpr int STATIC_MAX_DEVICES = 64;
static void* g_static_build_ptr[STATIC_MAX_DEVICES];
static std::mutex g_static_build_mu;

static int static_build_region(tacaw_ctx* ctx, void** out) {
    if (ctx->device < 0 || ctx->device >= STATIC_MAX_DEVICES)
        return fail(ctx, TACAW_E_UNSUPPORTED, "tacaw_build_slices_static: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_static_build_mu);
    if (!g_static_build_ptr[ctx->device]) {
        void* p = nullptr;
        TACAW_CUDA(ctx, cudaGetSymbolAddress(&p, g_static_build));
        if (!p) return fail(ctx, TACAW_E_CUDA, "tacaw_build_slices_static: cudaGetSymbolAddress returned a null address");
        g_static_build_ptr[ctx->device] = p;
    }
    *out = g_static_build_ptr[ctx->device];
    return TACAW_OK;
}

int launch_potential_static(tacaw_ctx* ctx, const double* d_pos, const int32_t* d_species, int natoms, int nframes, int nspecies,
                            const AbTable& ab, double dz, int nslices, double z0, float2* d_V, cudaStream_t st) {
    const int nx = ctx->grid.nx, ny = ctx->grid.ny;
    const long long ntotal = (long long)natoms * nframes;
    const long long nkeys_ll = (long long)nframes * nslices * nspecies;
    // same layout as the build region of the workspace: clamp counter (256 B) | keys ux uy sx sy [nt] | counts | offsets
    const long long nt_ll = ntotal > 0 ? ntotal : 1;
    const long long need = 256 + (long long)sizeof(int) * (5 * nt_ll + 2 * nkeys_ll + 2);
    if (ntotal > (1LL << 31) - 1 || nkeys_ll > (1LL << 30) || need > (long long)TACAW_STATIC_SCRATCH_BYTES)
        return fail(ctx, TACAW_E_UNSUPPORTED,
                    "tacaw_build_slices_static: this call needs " + std::to_string(need) + " bytes of scratch (256 + 4*(5*natoms*nframes + "
                    "2*nframes*nslices*nspecies + 2)), the static array holds " + std::to_string((long long)TACAW_STATIC_SCRATCH_BYTES) +
                    ": use tacaw_build_slices with a workspace");
    void* reg = nullptr;
    int rc = static_build_region(ctx, &reg);
    if (rc) return rc;
    const int nkeys = (int)nkeys_ll;
    const size_t nt = (size_t)nt_ll;
    int* d_nclamped = (int*)reg;
    int* keys = (int*)((char*)reg + 256);
    uint32_t* ux = (uint32_t*)(keys + nt);
    uint32_t* uy = ux + nt;
    uint32_t* sx = uy + nt;
    uint32_t* sy = sx + nt;
    int* counts = (int*)(sy + nt);
    int* offsets = counts + nkeys;
    // what must start at zero: the per-key counts (atomicAdd targets), the offsets, the clamp counter
    TACAW_CUDA(ctx, cudaMemsetAsync(counts, 0, sizeof(int) * (2 * (size_t)nkeys + 1), st));
    TACAW_CUDA(ctx, cudaMemsetAsync(d_nclamped, 0, sizeof(int), st));
    if (ntotal == 0) TACAW_CUDA(ctx, cudaMemsetAsync(d_V, 0, sizeof(float2) * (size_t)nframes * nslices * nx * ny, st));
    if (ntotal > 0) {
        k_atom_keys<<<(unsigned)((ntotal + 255) / 256), 256, 0, st>>>(d_pos, d_species, natoms, ntotal, nspecies, dz, nslices,
                                                                     z0, 1.0 / ctx->grid.lx_A, 1.0 / ctx->grid.ly_A, keys, ux,
                                                                     uy, counts, d_nclamped, ctx->d_flags);
        ctx->launches++;
    }
    k_scan_counts<<<1, 1024, 0, st>>>(counts, nkeys, offsets);
    ctx->launches++;
    if (ntotal > 0) {
        k_compact<<<(unsigned)(((long long)nkeys * 32 + 255) / 256), 256, 0, st>>>(keys, natoms, nslices * nspecies, nkeys, offsets,
                                                                                  ux, uy, sx, sy);
        ctx->launches++;
        const int hmax = ctx->hmax_pot;
        const int total_slices = nframes * nslices;
        static const bool use_tc = [] { const char* e = getenv("TACAW_K1_TC"); return e ? atoi(e) != 0 : true; }();
        if (use_tc && nspecies <= potential_tc_max_species())
            return launch_potential_tc(ctx, sx, sy, offsets, nspecies, ab, total_slices, d_V, st);
        for (int z0i = 0; z0i < total_slices; z0i += 65535) {
            int nz = total_slices - z0i < 65535 ? total_slices - z0i : 65535;
            dim3 grid((hmax + 1 + POT_T - 1) / POT_T, (ctx->kmaxmax_pot + 1 + POT_T - 1) / POT_T, nz);
            k_potential<<<grid, POT_THREADS, 0, st>>>(sx, sy, offsets + (size_t)z0i * nspecies, nspecies, ab, ctx->d_kmax_pot, hmax, nx,
                                              ny, (float)(1.0 / ctx->grid.lx_A), (float)(1.0 / ctx->grid.ly_A),
                                              d_V + (size_t)z0i * nx * ny);
            ctx->launches++;
        }
    }
    TACAW_CUDA(ctx, cudaGetLastError());
    return TACAW_OK;
}

// ---------------------------------------------------------------------------------------- K3
// Psi0[h,k] = amp * exp(-2 pi i (h xp/lx + k yp/ly)) inside the aperture, else 0 (q space).
// The aperture decision (lambda^2 q^2 <= alpha^2) is taken on the host in fp64 and arrives as
// kap[ix] = largest |k| inside the aperture for column ix (-1: none).
__global__ void k_probe_fill(const uint32_t* __restrict__ uxy, int nx, int ny, const int* __restrict__ kap, float amp,
                             float2* __restrict__ waves) {
    const int p = blockIdx.y;
    const size_t npix = (size_t)nx * ny;
    const uint32_t ux = uxy[2 * p], uy = uxy[2 * p + 1];
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < npix; i += (size_t)gridDim.x * blockDim.x) {
        int ix = (int)(i % nx), iy = (int)(i / nx);
        int h = ix < nx / 2 ? ix : ix - nx, k = iy < ny / 2 ? iy : iy - ny;
        float2 v = make_float2(0.f, 0.f);
        if (abs(k) <= kap[ix]) {
            float2 e = phase_fixed(ux, h), f = phase_fixed(uy, k);
            v = make_float2(amp * (e.x * f.x - e.y * f.y), amp * (e.x * f.y + e.y * f.x));
        }
        waves[(size_t)p * npix + i] = v;
    }
}

int launch_probe_fill(tacaw_ctx* ctx, const uint32_t* d_uxy, int nprobes, const int* d_kap, float amp, float2* d_waves,
                      cudaStream_t st) {
    const int nx = ctx->grid.nx, ny = ctx->grid.ny;
    int bx = (int)(((size_t)nx * ny + 255) / 256);
    if (bx > 1024) bx = 1024;
    k_probe_fill<<<dim3(bx, nprobes), 256, 0, st>>>(d_uxy, nx, ny, d_kap, amp, d_waves);
    ctx->launches++;
    TACAW_CUDA(ctx, cudaGetLastError());
    return TACAW_OK;
}

// ---------------------------------------------------------------------------------------- K5
__global__ void k_gather(const float2* __restrict__ q, const int* __restrict__ wp, const int* __restrict__ wf,
                         const int* __restrict__ idx, long long nroi, float2* __restrict__ buf, int nframes,
                         size_t npix, float scale) {
    const int w = blockIdx.y;
    const float2* src = q + (size_t)w * npix;
    float2* dst = buf + ((size_t)wp[w] * nframes + wf[w]) * (size_t)nroi;
    for (long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x; r < nroi; r += (long long)gridDim.x * blockDim.x) {
        float2 v = src[idx[r]];
        dst[r] = make_float2(v.x * scale, v.y * scale);
    }
}

// inverse ROI map for the fused gather: inv[pixel] = position in the ROI list, -1 elsewhere
__global__ void k_fill_int(int* __restrict__ p, long long n, int v) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) p[i] = v;
}
__global__ void k_roi_scatter(const int* __restrict__ idx, long long nroi, int* __restrict__ inv) {
    for (long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x; r < nroi; r += (long long)gridDim.x * blockDim.x) inv[idx[r]] = (int)r;
}
int launch_roi_inverse(tacaw_ctx* ctx, const int* d_idx, int64_t nroi, int* d_inv, cudaStream_t st) {
    const long long npix = (long long)ctx->grid.nx * ctx->grid.ny;
    k_fill_int<<<(unsigned)std::min<long long>((npix + 255) / 256, 4096), 256, 0, st>>>(d_inv, npix, -1);
    ctx->launches++;
    if (nroi > 0) {
        k_roi_scatter<<<(unsigned)std::min<long long>((nroi + 255) / 256, 4096), 256, 0, st>>>(d_idx, (long long)nroi, d_inv);
        ctx->launches++;
    }
    TACAW_CUDA(ctx, cudaGetLastError());
    return TACAW_OK;
}
// buffer rows of the waves about to be gathered: ROI pixels in columns outside the band limit are exactly zero and are
// never touched by the column kernel
__global__ void k_zero_slots(float2* __restrict__ buf, const int* __restrict__ slot, long long nroi) {
    float2* dst = buf + (size_t)slot[blockIdx.y] * (size_t)nroi;
    for (long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x; r < nroi; r += (long long)gridDim.x * blockDim.x)
        dst[r] = make_float2(0.f, 0.f);
}
int launch_zero_slots(tacaw_ctx* ctx, float2* d_buf, const int* d_slot, int nwaves, int64_t nroi, cudaStream_t st) {
    if (nwaves <= 0 || nroi <= 0) return TACAW_OK;
    int bx = (int)((nroi + 255) / 256);
    if (bx > 64) bx = 64;
    for (int w0 = 0; w0 < nwaves; w0 += 32768) {
        const int nw = nwaves - w0 < 32768 ? nwaves - w0 : 32768;
        k_zero_slots<<<dim3(bx, nw), 256, 0, st>>>(d_buf, d_slot + w0, (long long)nroi);
        ctx->launches++;
    }
    TACAW_CUDA(ctx, cudaGetLastError());
    return TACAW_OK;
}

int launch_gather(tacaw_ctx* ctx, const float2* d_q, int nwaves, const int* d_wp, const int* d_wf, const int* d_idx,
                  int64_t nroi, float2* d_buf, int nprobes, int nframes, cudaStream_t st) {
    (void)nprobes;
    if (nwaves <= 0 || nroi <= 0) return TACAW_OK;
    const size_t npix = (size_t)ctx->grid.nx * ctx->grid.ny;
    int bx = (int)((nroi + 255) / 256);
    if (bx > 64) bx = 64;
    for (int w0 = 0; w0 < nwaves; w0 += 32768) {
        int nw = nwaves - w0 < 32768 ? nwaves - w0 : 32768;
        k_gather<<<dim3(bx, nw), 256, 0, st>>>(d_q + (size_t)w0 * npix, d_wp + w0, d_wf + w0, d_idx, (long long)nroi, d_buf,
                                               nframes, npix, (float)(1.0 / sqrt((double)npix)));
        ctx->launches++;
    }
    TACAW_CUDA(ctx, cudaGetLastError());
    return TACAW_OK;
}

}  // namespace tacaw

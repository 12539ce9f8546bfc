// api.cu -- extern "C" entry points of libtacaw (see include/tacaw.h for the contract).
// Host logic only: argument checks, fp64 table generation, scratch management, launch order.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "ctx.h"
#include "fft2.cuh"

namespace tacaw {

int fail(tacaw_ctx* ctx, int code, const std::string& msg) {
    if (ctx) ctx->err = msg;
    return code;
}

int cuda_fail(tacaw_ctx* ctx, cudaError_t e, const char* where) {
    if (ctx) ctx->err = std::string("CUDA error: ") + cudaGetErrorString(e) + " at " + where;
    return TACAW_E_CUDA;
}

int region(tacaw_ctx* ctx, int r, size_t need, void** out, const char* who) {
    if (need == 0) { *out = ctx->d_ws ? ctx->d_ws + ctx->reg_off[r] : nullptr; return TACAW_OK; }
    if (!ctx->d_ws) return fail(ctx, TACAW_E_NOMEM, std::string(who) + ": no workspace set (tacaw_workspace_bytes / tacaw_set_workspace)");
    if (ctx->reg_bytes[r] < need)
        return fail(ctx, TACAW_E_NOMEM, std::string(who) + ": workspace region too small (" + std::to_string(ctx->reg_bytes[r]) + " < " +
                                            std::to_string(need) + " bytes): size it for this call with tacaw_workspace_bytes");
    *out = ctx->d_ws + ctx->reg_off[r];
    return TACAW_OK;
}

// Region sizes for the largest calls a caller announces (tacaw_sizes).  Every region is a multiple of 256 bytes.
static void region_sizes(const tacaw_ctx* ctx, const tacaw_sizes& z, size_t (&bytes)[tacaw_ctx::R_COUNT]) {
    auto up = [](size_t v) { return (v + 255) / 256 * 256; };
    const size_t natoms = (size_t)(z.natoms > 0 ? z.natoms : 0), nframes = (size_t)(z.nframes > 0 ? z.nframes : 0);
    const size_t nslices = (size_t)(z.nslices > 0 ? z.nslices : 0), nseg = (size_t)(z.nsegments > 0 ? z.nsegments : 1);
    const size_t nwaves = (size_t)(z.nwaves > 0 ? z.nwaves : 0), nprobes = (size_t)(z.nprobes > 0 ? z.nprobes : 0);
    const size_t nt = natoms * nframes > 0 ? natoms * nframes : 1, nkeys = nframes * nslices * MAX_SPECIES;
    // build_slices: clamp counter | keys ux uy sx sy [nt] | counts [nkeys] offsets [nkeys+1]
    bytes[tacaw_ctx::R_BUILD] = up(256 + sizeof(int) * (5 * nt + 2 * nkeys + 2));
    bytes[tacaw_ctx::R_STAGE] = z.host_staging ? up(sizeof(double) * 3 * natoms * nframes + sizeof(int32_t) * natoms + 64) : 0;
    bytes[tacaw_ctx::R_PROBE] = up(sizeof(int) * (size_t)ctx->grid.nx + sizeof(uint32_t) * 2 * nprobes + 64);
    // propagate: wave_frame | wave_probe | tuples (<= (nwaves + 64) * rpt) | transmission pointers
    const size_t rpt = ctx->generic_path ? 1 : (size_t)row_tuple_size(ctx->grid.nx);
    bytes[tacaw_ctx::R_PROP] = up(sizeof(int) * (3 * nwaves + (nwaves + 64) * rpt) + 16 + sizeof(void*) * nframes * nseg + 64);
    bytes[tacaw_ctx::R_ACC] = up(sizeof(int) * 2 * nwaves + 64);
    bytes[tacaw_ctx::R_SPEC] = up(SPEC_TABLE_BYTES);
}

// Two-half pinned arena: a half is reused only after the copies issued from it have completed (event), never by
// draining the device.
int upload(tacaw_ctx* ctx, void* dst, const void* src, size_t bytes, cudaStream_t st) {
    if (bytes == 0) return TACAW_OK;
    const size_t need = (bytes + 63) / 64 * 64;
    const size_t half = ctx->arena_bytes / 2;
    if (!ctx->h_arena || need > half) {   // pageable copy: staged by the runtime before it returns
        TACAW_CUDA(ctx, cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, st));
        return TACAW_OK;
    }
    int h = ctx->arena_off >= half ? 1 : 0;
    if (ctx->arena_off + need > (size_t)(h + 1) * half) {
        // leave this half: mark its copies with an event, enter the other half once ITS copies are done
        TACAW_CUDA(ctx, cudaEventRecord(ctx->ev_arena[h], st));
        ctx->arena_used[h] = true;
        h ^= 1;
        if (ctx->arena_used[h]) TACAW_CUDA(ctx, cudaEventSynchronize(ctx->ev_arena[h]));
        ctx->arena_off = (size_t)h * half;
    }
    char* hp = ctx->h_arena + ctx->arena_off;
    ctx->arena_off += need;
    memcpy(hp, src, bytes);
    TACAW_CUDA(ctx, cudaMemcpyAsync(dst, hp, bytes, cudaMemcpyHostToDevice, st));
    return TACAW_OK;
}

static inline int sgn_index(int i, int n) { return i < n / 2 ? i : i - n; }

// O5 mask predicate, restated from DESIGN.md (not shared with the oracle).
static bool mask_in_band(int h, int k, const tacaw_grid& g) {
    if (g.nx == g.ny && g.lx_A == g.ly_A) return 9LL * ((long long)h * h + (long long)k * k) <= (long long)g.nx * g.nx;
    double qx = h / g.lx_A, qy = k / g.ly_A;
    double qn = std::fmin(g.nx / (2.0 * g.lx_A), g.ny / (2.0 * g.ly_A));
    return qx * qx + qy * qy <= (4.0 / 9.0) * qn * qn;
}

// powers of two in [16, 2048] run on the register FFTs; other even sizes with prime factors 2, 3, 5, 7 on generic.cu
static bool supported_n(int n) { return (n >= 16 && n <= 2048 && (n & (n - 1)) == 0) || generic_grid_supported(n); }

// twiddle table of the slice-step transforms of length n (layout: fft2.cuh)
static void make_roots(int n, bool generic, std::vector<float2>& out) {
    if (generic) {                       // generic.cu: the n-th roots of unity
        out.resize(n);
        generic_host_table(n, out.data());
        return;
    }
    out.resize(slice_step_table_elems(n));
    slice_step_host_table(n, out.data());
}

static int ensure_propagator(tacaw_ctx* ctx, double dz, cudaStream_t st) {
    if (ctx->dz_cached == dz) return TACAW_OK;
    const tacaw_grid& g = ctx->grid;
    std::vector<float2> px(g.nx), py(g.ny);
    for (int ix = 0; ix < g.nx; ++ix) {
        double h = sgn_index(ix, g.nx);
        double ang = -M_PI * ctx->beam.lambda_A * dz * (h / g.lx_A) * (h / g.lx_A);
        px[ix] = make_float2((float)(std::cos(ang) / g.nx), (float)(std::sin(ang) / g.nx));
    }
    for (int iy = 0; iy < g.ny; ++iy) {
        double k = sgn_index(iy, g.ny);
        double ang = -M_PI * ctx->beam.lambda_A * dz * (k / g.ly_A) * (k / g.ly_A);
        py[iy] = make_float2((float)(std::cos(ang) / g.ny), (float)(std::sin(ang) / g.ny));
    }
    // stream-ordered: kernels already queued on `st` with the previous dz finish before the copy (a context is driven from
    // one stream at a time, tacaw.h)
    int rc = upload(ctx, ctx->d_px, px.data(), sizeof(float2) * g.nx, st);
    if (rc) return rc;
    if ((rc = upload(ctx, ctx->d_py, py.data(), sizeof(float2) * g.ny, st))) return rc;
    ctx->dz_cached = dz;
    return TACAW_OK;
}

}  // namespace tacaw

using namespace tacaw;

extern "C" {

const char* tacaw_version(void) { return "tacaw-b200 0.1 (sm_100a)"; }

const char* tacaw_last_error(const tacaw_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int64_t tacaw_launch_count(const tacaw_ctx* ctx) { return ctx ? ctx->launches : 0; }

int tacaw_create(tacaw_ctx** out, const tacaw_grid* grid, const tacaw_beam* beam, int device) {
    if (!out || !grid || !beam) return TACAW_E_ARG;
    *out = nullptr;
    if (!supported_n(grid->nx) || !supported_n(grid->ny)) return TACAW_E_UNSUPPORTED;
    if (!(grid->lx_A > 0) || !(grid->ly_A > 0) || !(beam->lambda_A > 0)) return TACAW_E_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0 || device < 0 || device >= ndev) {
        (void)cudaGetLastError();
        return TACAW_E_CUDA;
    }
    tacaw_ctx* ctx = new tacaw_ctx();
    ctx->grid = *grid;
    ctx->beam = *beam;
    ctx->device = device;
    DeviceGuard guard(ctx);           // the caller's current device is restored on return
    if (!guard.ok) { delete ctx; return TACAW_E_CUDA; }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) == cudaSuccess) {
        ctx->num_sms = prop.multiProcessorCount;
        ctx->l2_bytes = (size_t)prop.l2CacheSize;
    }
    const int nx = grid->nx, ny = grid->ny;
    // band-limit column extents (propagator) and potential extents (Nyquist excluded, reading G4)
    ctx->kmax.assign(nx, -1);
    ctx->kmax_pot.assign(nx, -1);
    ctx->hmax = 0;
    ctx->hmax_pot = 0;
    ctx->kmaxmax_pot = 0;
    // per column: the in-band k form an interval |k| <= km (the mask is a disc, monotone in |k|): bisect for km instead
    // of testing every cell.  Potential extents additionally exclude the Nyquist row and column (reading G4).
    for (int ix = 0; ix < nx; ++ix) {
        const int h = sgn_index(ix, nx);
        int km = -1;
        if (!beam->bandlimit) km = ny / 2;
        else if (mask_in_band(h, 0, *grid)) {
            int lo = 0, hi = ny / 2 + 1;              // invariant: in(lo), !in(hi) (k = ny/2 + 1 is outside any 2/3 disc)
            while (hi - lo > 1) {
                const int mid = (lo + hi) / 2;
                if (mid <= ny / 2 && mask_in_band(h, mid, *grid)) lo = mid; else hi = mid;
            }
            km = lo;
        }
        int kp = km;
        if (2 * kp >= ny) kp = (ny - 1) / 2;          // largest |k| below Nyquist
        if (2 * h == -nx) kp = -1;
        ctx->kmax[ix] = km;
        ctx->kmax_pot[ix] = kp;
        const int ah = h < 0 ? -h : h;
        if (km >= 0 && ah > ctx->hmax) ctx->hmax = ah;
        if (kp >= 0 && ah > ctx->hmax_pot) ctx->hmax_pot = ah;
        if (kp > ctx->kmaxmax_pot) ctx->kmaxmax_pot = kp;
        if (km > ctx->kmaxmax) ctx->kmaxmax = km;
    }
    std::vector<float2> rx, ry;
    const auto pow2 = [](int n) { return (n & (n - 1)) == 0; };
    ctx->generic_path = !pow2(nx) || !pow2(ny);       // one dimension off the powers of two puts both passes on generic.cu
    make_roots(nx, ctx->generic_path, rx);
    make_roots(ny, ctx->generic_path, ry);
    bool ok = cudaMalloc(&ctx->d_roots_x, sizeof(float2) * rx.size()) == cudaSuccess &&
              cudaMalloc(&ctx->d_roots_y, sizeof(float2) * ry.size()) == cudaSuccess &&
              cudaMalloc(&ctx->d_kmax, sizeof(int) * nx) == cudaSuccess &&
              cudaMalloc(&ctx->d_kmax_pot, sizeof(int) * nx) == cudaSuccess &&
              cudaMalloc(&ctx->d_px, sizeof(float2) * nx) == cudaSuccess &&
              cudaMalloc(&ctx->d_py, sizeof(float2) * ny) == cudaSuccess &&
              cudaMalloc(&ctx->d_flags, 4 * sizeof(int)) == cudaSuccess &&
              cudaMemset(ctx->d_flags, 0, 4 * sizeof(int)) == cudaSuccess;
    if (cudaMallocHost((void**)&ctx->h_arena, (size_t)8 << 20) == cudaSuccess) ctx->arena_bytes = (size_t)8 << 20;
    else { (void)cudaGetLastError(); ctx->h_arena = nullptr; }
    for (int i = 0; i < 2; ++i) ok = ok && cudaEventCreateWithFlags(&ctx->ev_arena[i], cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaMemcpy(ctx->d_roots_x, rx.data(), sizeof(float2) * rx.size(), cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemcpy(ctx->d_roots_y, ry.data(), sizeof(float2) * ry.size(), cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemcpy(ctx->d_kmax, ctx->kmax.data(), sizeof(int) * nx, cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemcpy(ctx->d_kmax_pot, ctx->kmax_pot.data(), sizeof(int) * nx, cudaMemcpyHostToDevice) == cudaSuccess;
    ok = ok && cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming) == cudaSuccess;
    for (int i = 0; i < tacaw_ctx::MAX_AUX; ++i)
        ok = ok && cudaStreamCreateWithFlags(&ctx->aux[i], cudaStreamNonBlocking) == cudaSuccess &&
             cudaEventCreateWithFlags(&ctx->ev_join[i], cudaEventDisableTiming) == cudaSuccess;
    if (!ok) {
        (void)cudaGetLastError();
        tacaw_destroy(ctx);
        return TACAW_E_CUDA;
    }
    *out = ctx;
    return TACAW_OK;
}

int tacaw_destroy(tacaw_ctx* ctx) {
    if (!ctx) return TACAW_E_ARG;
    {
        DeviceGuard guard(ctx);
        cudaDeviceSynchronize();
        cudaFree(ctx->d_roots_x); cudaFree(ctx->d_roots_y); cudaFree(ctx->d_kmax); cudaFree(ctx->d_kmax_pot);
        cudaFree(ctx->d_px); cudaFree(ctx->d_py); cudaFree(ctx->d_flags);      // the workspace is the caller's
        if (ctx->h_arena) cudaFreeHost(ctx->h_arena);
        for (int i = 0; i < 2; ++i)
            if (ctx->ev_arena[i]) cudaEventDestroy(ctx->ev_arena[i]);
        for (int i = 0; i < tacaw_ctx::MAX_AUX; ++i) {
            if (ctx->aux[i]) cudaStreamDestroy(ctx->aux[i]);
            if (ctx->ev_join[i]) cudaEventDestroy(ctx->ev_join[i]);
        }
        if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
        (void)cudaGetLastError();
    }
    delete ctx;
    return TACAW_OK;
}

size_t tacaw_workspace_bytes(const tacaw_ctx* ctx, const tacaw_sizes* sizes) {
    if (!ctx || !sizes) return 0;
    size_t b[tacaw_ctx::R_COUNT];
    region_sizes(ctx, *sizes, b);
    size_t tot = 0;
    for (int r = 0; r < tacaw_ctx::R_COUNT; ++r) tot += b[r];
    return tot;
}

int tacaw_set_workspace(tacaw_ctx* ctx, void* d_workspace, size_t bytes, const tacaw_sizes* sizes) {
    TACAW_ENTER(ctx);
    if (!sizes || (!d_workspace && bytes > 0)) return fail(ctx, TACAW_E_ARG, "tacaw_set_workspace: bad argument");
    if (((uintptr_t)d_workspace & 255) != 0) return fail(ctx, TACAW_E_ARG, "tacaw_set_workspace: the workspace must be 256-byte aligned");
    size_t b[tacaw_ctx::R_COUNT];
    region_sizes(ctx, *sizes, b);
    size_t tot = 0;
    for (int r = 0; r < tacaw_ctx::R_COUNT; ++r) tot += b[r];
    if (bytes < tot) return fail(ctx, TACAW_E_NOMEM, "tacaw_set_workspace: " + std::to_string(bytes) + " bytes given, " + std::to_string(tot) + " needed for these sizes");
    ctx->d_ws = (char*)d_workspace;
    ctx->ws_bytes = bytes;
    size_t off = 0;
    for (int r = 0; r < tacaw_ctx::R_COUNT; ++r) { ctx->reg_off[r] = off; ctx->reg_bytes[r] = b[r]; off += b[r]; }
    ctx->maps.clear();
    return TACAW_OK;
}

int tacaw_device_status(tacaw_ctx* ctx, void* stream) {
    TACAW_ENTER(ctx);
    int h[4] = {0, 0, 0, 0};
    TACAW_CUDA(ctx, cudaMemcpyAsync(h, ctx->d_flags, sizeof(h), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    TACAW_CUDA(ctx, cudaStreamSynchronize((cudaStream_t)stream));
    if (h[0] > 0) {
        TACAW_CUDA(ctx, cudaMemsetAsync(ctx->d_flags, 0, sizeof(h), (cudaStream_t)stream));
        return fail(ctx, TACAW_E_ARG, "tacaw_build_slices: " + std::to_string(h[0]) + " species id(s) out of range since the last status check");
    }
    return TACAW_OK;
}

int tacaw_build_slices(tacaw_ctx* ctx, const double* d_pos_A, const int32_t* d_species, int natoms, int nframes,
                       const tacaw_species* species, double dz, int nslices, double z0, void* d_trans, int* n_clamped,
                       void* stream) {
    TACAW_ENTER(ctx);
    if (nframes == 0) { if (n_clamped) *n_clamped = 0; return TACAW_OK; }
    if (natoms < 0 || nframes < 0 || nslices <= 0 || !(dz > 0) || !d_trans || !species || species->nspecies <= 0 || !species->a ||
        !species->b || (natoms > 0 && (!d_pos_A || !d_species)))
        return fail(ctx, TACAW_E_ARG, "tacaw_build_slices: bad argument");
    cudaStream_t st = (cudaStream_t)stream;
    const int ns = species->nspecies;
    const int nx = ctx->grid.nx, ny = ctx->grid.ny;
    if (ns > MAX_SPECIES) return fail(ctx, TACAW_E_UNSUPPORTED, "tacaw_build_slices: at most 8 species");
    AbTable ab{};
    for (int s = 0; s < ns; ++s)
        for (int i = 0; i < 4; ++i) {
            ab.a[s][i] = (float)species->a[4 * s + i];
            ab.b[s][i] = (float)species->b[4 * s + i];
        }
    int* d_ncl = nullptr;             // clamped atoms of this call (first word of the build region)
    int rc = launch_potential(ctx, d_pos_A, d_species, natoms, nframes, ns, ab, dz, nslices, z0, (float2*)d_trans, &d_ncl, st);
    if (rc) return rc;
    // V(q) -> v(r) -> t = exp(i sigma v):  IFFT_y over the in-band columns, then IFFT_x + exp per row
    ColArgs ca{};
    ca.waves = (float2*)d_trans; ca.nwaves = nframes * nslices; ca.nx = nx; ca.hmax = ctx->hmax_pot; ca.roots = ctx->d_roots_y;
    ca.px = nullptr; ca.py = nullptr; ca.kmax = ctx->d_kmax_pot; ca.pscale = 1.f; ca.kmaxmax = -1;
    rc = launch_col(ctx, COL_INV, ca, ny, st);
    if (rc) return rc;
    RowArgs ra{};
    ra.waves = (float2*)d_trans; ra.nwaves = nframes * nslices; ra.ny = ny; ra.hmax = ctx->hmax_pot; ra.roots = ctx->d_roots_x;
    ra.scale = (float)(ctx->beam.sigma_rad_per_VA / (ctx->grid.lx_A * ctx->grid.ly_A));
    rc = launch_row(ctx, ROW_TRANS, ra, st);
    if (rc) return rc;
    if (n_clamped) {
        // the one synchronising path: also reports (and clears) the sticky species-id flag
        int h_ncl = 0;
        TACAW_CUDA(ctx, cudaMemcpyAsync(&h_ncl, d_ncl, sizeof(int), cudaMemcpyDeviceToHost, st));
        TACAW_CUDA(ctx, cudaStreamSynchronize(st));
        *n_clamped = h_ncl;
        return tacaw_device_status(ctx, stream);
    }
    return TACAW_OK;
}

int tacaw_build_slices_static(tacaw_ctx* ctx, const double* d_pos_A, const int32_t* d_species, int natoms, int nframes,
                              const tacaw_species* species, double dz, int nslices, double z0, void* d_trans, void* stream) {
    TACAW_ENTER(ctx);
    if (nframes == 0) return TACAW_OK;
    if (natoms < 0 || nframes < 0 || nslices <= 0 || !(dz > 0) || !d_trans || !species || species->nspecies <= 0 || !species->a ||
        !species->b || (natoms > 0 && (!d_pos_A || !d_species)))
        return fail(ctx, TACAW_E_ARG, "tacaw_build_slices_static: bad argument");
    cudaStream_t st = (cudaStream_t)stream;
    const int ns = species->nspecies;
    const int nx = ctx->grid.nx, ny = ctx->grid.ny;
    if (ns > MAX_SPECIES) return fail(ctx, TACAW_E_UNSUPPORTED, "tacaw_build_slices_static: at most 8 species");
    AbTable ab{};
    for (int s = 0; s < ns; ++s)
        for (int i = 0; i < 4; ++i) {
            ab.a[s][i] = (float)species->a[4 * s + i];
            ab.b[s][i] = (float)species->b[4 * s + i];
        }
    // sizes beyond the static array are refused before anything is queued
    int rc = launch_potential_static(ctx, d_pos_A, d_species, natoms, nframes, ns, ab, dz, nslices, z0, (float2*)d_trans, st);
    if (rc) return rc;
    // V(q) -> v(r) -> t = exp(i sigma v), as in tacaw_build_slices (these two kernels use no scratch)
    ColArgs ca{};
    ca.waves = (float2*)d_trans; ca.nwaves = nframes * nslices; ca.nx = nx; ca.hmax = ctx->hmax_pot; ca.roots = ctx->d_roots_y;
    ca.px = nullptr; ca.py = nullptr; ca.kmax = ctx->d_kmax_pot; ca.pscale = 1.f; ca.kmaxmax = -1;
    rc = launch_col(ctx, COL_INV, ca, ny, st);
    if (rc) return rc;
    RowArgs ra{};
    ra.waves = (float2*)d_trans; ra.nwaves = nframes * nslices; ra.ny = ny; ra.hmax = ctx->hmax_pot; ra.roots = ctx->d_roots_x;
    ra.scale = (float)(ctx->beam.sigma_rad_per_VA / (ctx->grid.lx_A * ctx->grid.ly_A));
    return launch_row(ctx, ROW_TRANS, ra, st);
}

int tacaw_build_slices_host(tacaw_ctx* ctx, const double* h_pos_A, const int32_t* h_species, int natoms, int nframes,
                            const tacaw_species* species, double dz, int nslices, double z0, void* d_trans,
                            int* n_clamped, void* stream) {
    TACAW_ENTER(ctx);
    if (natoms < 0 || nframes < 0 || !species || (natoms > 0 && nframes > 0 && (!h_pos_A || !h_species))) return fail(ctx, TACAW_E_ARG, "bad argument");
    // species ids are on the host here: validate them before anything is queued
    for (int j = 0; j < natoms; ++j)
        if (h_species[j] < 0 || h_species[j] >= species->nspecies) return fail(ctx, TACAW_E_ARG, "tacaw_build_slices_host: species id out of range");
    cudaStream_t st = (cudaStream_t)stream;
    size_t nb_pos = sizeof(double) * 3 * (size_t)natoms * (size_t)nframes, nb_sp = sizeof(int32_t) * (size_t)natoms;
    void* stage = nullptr;
    int rc = region(ctx, tacaw_ctx::R_STAGE, nb_pos + nb_sp + 64, &stage, "tacaw_build_slices_host");
    if (rc) return rc;
    double* d_pos = (double*)stage;
    int32_t* d_sp = (int32_t*)((char*)stage + nb_pos);
    if (natoms > 0 && nframes > 0) {
        TACAW_CUDA(ctx, cudaMemcpyAsync(d_pos, h_pos_A, nb_pos, cudaMemcpyHostToDevice, st));
        TACAW_CUDA(ctx, cudaMemcpyAsync(d_sp, h_species, nb_sp, cudaMemcpyHostToDevice, st));
    }
    // n_clamped == NULL: nothing to read back, the call stays asynchronous (pinned sources; pageable ones are staged by
    // the runtime before cudaMemcpyAsync returns)
    return tacaw_build_slices(ctx, d_pos, d_sp, natoms, nframes, species, dz, nslices, z0, d_trans, n_clamped, stream);
}

int tacaw_make_probes(tacaw_ctx* ctx, const double* probe_xy_A, int nprobes, double alpha_rad, void* d_waves,
                      void* stream) {
    TACAW_ENTER(ctx);
    if (nprobes < 0 || (nprobes > 0 && (!probe_xy_A || !d_waves)) || alpha_rad < 0)
        return fail(ctx, TACAW_E_ARG, "tacaw_make_probes: bad argument");
    if (nprobes == 0) return TACAW_OK;
    cudaStream_t st = (cudaStream_t)stream;
    const tacaw_grid& g = ctx->grid;
    const int nx = g.nx, ny = g.ny;
    // aperture decision in fp64 (O4, reading G8): A = 1 iff lambda^2 q^2 <= alpha^2
    std::vector<int> kap(nx, -1);
    long long n_in = 0;
    int hap = 0;
    const double lam = ctx->beam.lambda_A;
    for (int ix = 0; ix < nx; ++ix) {
        int h = sgn_index(ix, nx);
        for (int iy = 0; iy < ny; ++iy) {
            int k = sgn_index(iy, ny);
            double q2 = (h / g.lx_A) * (h / g.lx_A) + (k / g.ly_A) * (k / g.ly_A);
            if (lam * lam * q2 <= alpha_rad * alpha_rad) {
                ++n_in;
                int ak = k < 0 ? -k : k;
                // the disc is symmetric except for the unpaired Nyquist index -ny/2
                if (2 * ak < ny && ak > kap[ix]) kap[ix] = ak;
                if (2 * ak == ny) return fail(ctx, TACAW_E_UNSUPPORTED, "aperture reaches the Nyquist frequency");
                int ah = h < 0 ? -h : h;
                if (ah > hap) hap = ah;
            }
        }
    }
    if (n_in == 0) return fail(ctx, TACAW_E_ARG, "empty aperture");
    std::vector<uint32_t> uxy(2 * (size_t)nprobes);
    for (int p = 0; p < nprobes; ++p) {
        double fx = probe_xy_A[2 * p] / g.lx_A, fy = probe_xy_A[2 * p + 1] / g.ly_A;
        fx -= std::floor(fx);
        fy -= std::floor(fy);
        uxy[2 * p] = (uint32_t)(unsigned long long)std::llrint(fx * 4294967296.0);
        uxy[2 * p + 1] = (uint32_t)(unsigned long long)std::llrint(fy * 4294967296.0);
    }
    size_t need = sizeof(int) * nx + sizeof(uint32_t) * uxy.size() + 64;
    void* reg = nullptr;
    int rc = region(ctx, tacaw_ctx::R_PROBE, need, &reg, "tacaw_make_probes");
    if (rc) return rc;
    int* d_kap = (int*)reg;
    uint32_t* d_uxy = (uint32_t*)(d_kap + nx);
    if ((rc = upload(ctx, d_kap, kap.data(), sizeof(int) * nx, st))) return rc;
    if ((rc = upload(ctx, d_uxy, uxy.data(), sizeof(uint32_t) * uxy.size(), st))) return rc;
    // unit norm: the unscaled inverse transform of n_in unit phasors has sum |psi|^2 = nx ny n_in
    float amp = (float)(1.0 / std::sqrt((double)nx * (double)ny * (double)n_in));
    rc = launch_probe_fill(ctx, d_uxy, nprobes, d_kap, amp, (float2*)d_waves, st);
    if (rc) return rc;
    ColArgs ca{};
    ca.waves = (float2*)d_waves; ca.nwaves = nprobes; ca.nx = nx; ca.hmax = hap; ca.roots = ctx->d_roots_y;
    ca.kmax = d_kap; ca.pscale = 1.f; ca.kmaxmax = -1;
    rc = launch_col(ctx, COL_INV, ca, ny, st);
    if (rc) return rc;
    RowArgs ra{};
    ra.waves = (float2*)d_waves; ra.nwaves = nprobes; ra.ny = ny; ra.hmax = hap; ra.roots = ctx->d_roots_x;
    rc = launch_row(ctx, ROW_LAST, ra, st);
    if (rc) return rc;
    // the probe region is private to this entry point and reuse is stream-ordered: no synchronisation
    return TACAW_OK;
}

// fused gather (a6) of tacaw_propagate_accumulate: where the last column kernel puts the ROI pixels
struct GatherTarget {
    const int32_t* wave_time;      // HOST [nwaves] frame index on the buffer's time axis
    const int* d_roi_inv;          // DEVICE [ny][nx]
    int64_t nroi;
    float2* d_buf;
    int nprobes_buf, nframes_buf;
};

static int propagate_impl(tacaw_ctx* ctx, void* d_waves, const void* d_probes, int nprobes, const int32_t* wave_probe,
                          const int32_t* wave_frame, int nwaves, const void* const* d_trans, int nframes,
                          const int32_t* nslices_per_segment, int nsegments, double dz, int output_space, const GatherTarget* gt,
                          void* stream) {
    if (nwaves < 0 || nframes <= 0 || nsegments <= 0 || !(dz > 0) || !d_trans || !nslices_per_segment ||
        (nwaves > 0 && (!d_waves || !wave_frame)) || (d_probes && (!wave_probe || nprobes <= 0)) ||
        (output_space != 0 && output_space != 1))
        return fail(ctx, TACAW_E_ARG, "tacaw_propagate: bad argument");
    if (nwaves == 0) return TACAW_OK;
    int total = 0;
    for (int k = 0; k < nsegments; ++k) {
        if (nslices_per_segment[k] < 0) return fail(ctx, TACAW_E_ARG, "negative slice count");
        total += nslices_per_segment[k];
    }
    if (total == 0) return fail(ctx, TACAW_E_ARG, "tacaw_propagate: no slices");
    for (int w = 0; w < nwaves; ++w) {
        if (wave_frame[w] < 0 || wave_frame[w] >= nframes) return fail(ctx, TACAW_E_ARG, "wave_frame out of range");
        if (d_probes && (wave_probe[w] < 0 || wave_probe[w] >= nprobes)) return fail(ctx, TACAW_E_ARG, "wave_probe out of range");
    }
    for (int i = 0; i < nframes * nsegments; ++i)
        if (!d_trans[i] && nslices_per_segment[i % nsegments] > 0) return fail(ctx, TACAW_E_ARG, "null transmission pointer");
    cudaStream_t st = (cudaStream_t)stream;
    int rc = ensure_propagator(ctx, dz, st);
    if (rc) return rc;
    const tacaw_grid& g = ctx->grid;
    const size_t npix = (size_t)g.nx * g.ny;
    // metadata: [wave_frame nwaves][wave_probe nwaves][wave_slot nwaves][tuples <= nwaves*rpt][trans ptrs nframes*nseg]
    const int rpt = ctx->generic_path ? 1 : row_tuple_size(g.nx);
    size_t nb_i = sizeof(int) * (size_t)nwaves;
    size_t nb_t = sizeof(int) * ((size_t)nwaves + 64) * rpt;
    size_t off_t = 3 * nb_i;
    size_t off_p = ((off_t + nb_t + 15) / 16) * 16;
    size_t need = off_p + sizeof(void*) * (size_t)nframes * nsegments + 64;
    void* meta = nullptr;
    rc = region(ctx, tacaw_ctx::R_PROP, need, &meta, "tacaw_propagate");
    if (rc) return rc;
    int* d_wf = (int*)meta;
    int* d_wp = d_wf + nwaves;
    int* d_ws = d_wp + nwaves;
    int* d_tup = (int*)((char*)meta + off_t);
    const float2** d_tp = (const float2**)((char*)meta + off_p);
    if ((rc = upload(ctx, d_wf, wave_frame, nb_i, st))) return rc;
    if (d_probes && (rc = upload(ctx, d_wp, wave_probe, nb_i, st))) return rc;
    if ((rc = upload(ctx, (void*)d_tp, d_trans, sizeof(void*) * (size_t)nframes * nsegments, st))) return rc;
    if (gt) {
        std::vector<int> slot(nwaves);
        for (int w = 0; w < nwaves; ++w) slot[w] = wave_probe[w] * gt->nframes_buf + gt->wave_time[w];
        if ((rc = upload(ctx, d_ws, slot.data(), nb_i, st))) return rc;
        // ROI pixels outside the band limit are exactly zero and no column launch reaches them
        if ((rc = launch_zero_slots(ctx, gt->d_buf, d_ws, nwaves, gt->nroi, st))) return rc;
    }

    // depth-first over groups of waves small enough to stay L2-resident between the two kernels of
    // a slice step: all slices for group 0, then group 1, ...
    // a few groups are in flight at once (one per stream)
    // Defaults swept on B200 (fraction of the roofline; round 2, with the board at its 1 kW power cap the schedules that keep
    // more in flight lose SM clock): 512^2, 3 streams: 20 MB 0.533, 25 MB 0.552, 29 MB 0.562, 34 MB 0.563, 42 MB 0.535;
    // 4 streams lower everywhere.  1024^2 (waves per group, 2 / 3 / 4 streams): 3: 0.468 / 0.485 / 0.470, 5: 0.493 / 0.467 /
    // 0.440, 6: 0.494 / 0.462 / 0.454.  2048^2: see below.
    size_t budget = ctx->l2_bytes ? (size_t)(ctx->l2_bytes / 4.2) : (size_t)30 << 20;
    int gmin = 3;
    bool tuned = true;
    if (const char* e = getenv("TACAW_L2_GROUP_MB")) {
        double mb = atof(e);
        if (mb > 0) {
            budget = (size_t)(mb * 1048576.0);
            gmin = 1;
            tuned = false;
        }
    }
    const size_t wave_bytes = npix * sizeof(float2);
    int gmax = (int)(budget / wave_bytes);
    if (gmax >= 2 * rpt) gmax -= gmax % rpt;      // whole row tuples: a short tuple repeats its last wave (wasted work)
    // A wave larger than the budget (2048^2: 33.6 MB, 22.4 MB in band): what stays L2-resident is the TOTAL in flight, and
    // beyond ~90 MB of in-band waves plus the streaming t_n slice (33.6 MB) the 126 MB L2 thrashes.  Swept on B200 (streams x
    // waves per group, fraction of the roofline): 1x3 0.326, 2x2 0.346, 2x3 0.333, 3x2 0.326, 3x3 0.331, any x4 0.27-0.28.
    const bool huge = tuned && gmax < 2;
    const bool large = tuned && !huge && wave_bytes >= ((size_t)8 << 20);      // 1024^2: two streams x five waves
    if (huge) gmax = 2;
    else if (large) gmax = 5;
    else if (gmax < gmin) gmax = gmin;
    const int ngroups = (nwaves + gmax - 1) / gmax;
    static const int env_streams = [] {
        const char* e = getenv("TACAW_STREAMS");
        int v = e ? atoi(e) : 0;
        return v < 0 ? 0 : (v > 1 + tacaw_ctx::MAX_AUX ? 1 + tacaw_ctx::MAX_AUX : v);
    }();
    const int max_streams = env_streams ? env_streams : ((huge || large) ? 2 : 3);
    const int nstreams = ngroups < max_streams ? ngroups : max_streams;
    const bool fork = nstreams >= 2;
    cudaStream_t user_st = st;
    // group boundaries (balanced; a boundary moves to the nearest frame change within a quarter group) and the
    // wave tuples of every group: runs of up to `rpt` consecutive waves of the same frame, indices relative to the
    // group; a short tuple repeats its last wave
    std::vector<int> gw(ngroups + 1, 0), tup, tup_off(ngroups + 1, 0);
    for (int gi = 0; gi < ngroups; ++gi) {
        const int w0 = gw[gi];
        int w1 = (int)(((long long)(gi + 1) * nwaves) / ngroups);
        if (gi + 1 < ngroups) {
            const int slack = (w1 - w0) / 4;
            for (int d = 0; d <= slack; ++d) {
                if (w1 + d < nwaves && wave_frame[w1 + d] != wave_frame[w1 + d - 1]) { w1 += d; break; }
                if (w1 - d > w0 && wave_frame[w1 - d] != wave_frame[w1 - d - 1]) { w1 -= d; break; }
            }
            if (w1 < w0) w1 = w0;
        } else {
            w1 = nwaves;
        }
        gw[gi + 1] = w1;
        for (int w = w0; w < w1;) {
            int e = w + 1;
            while (e < w1 && e - w < rpt && wave_frame[e] == wave_frame[w]) ++e;
            for (int r = 0; r < rpt; ++r) tup.push_back((w + r < e ? w + r : e - 1) - w0);
            w = e;
        }
        tup_off[gi + 1] = (int)(tup.size() / rpt);
    }
    if (!tup.empty() && (rc = upload(ctx, d_tup, tup.data(), sizeof(int) * tup.size(), user_st))) return rc;
    if (fork) {
        TACAW_CUDA(ctx, cudaEventRecord(ctx->ev_fork, user_st));
        for (int i = 0; i + 1 < nstreams; ++i) TACAW_CUDA(ctx, cudaStreamWaitEvent(ctx->aux[i], ctx->ev_fork, 0));
    }
    for (int gi = 0; gi < ngroups; ++gi) {
        st = (gi % nstreams) ? ctx->aux[gi % nstreams - 1] : user_st;
        const int w0 = gw[gi], w1 = gw[gi + 1];
        const int nw = w1 - w0;
        if (nw <= 0) continue;
        int step = 0;
        for (int k = 0; k < nsegments; ++k) {
            for (int n = 0; n < nslices_per_segment[k]; ++n, ++step) {
                RowArgs ra{};
                ra.waves = (float2*)d_waves + (size_t)w0 * npix;
                ra.probes = (step == 0) ? (const float2*)d_probes : nullptr;
                ra.wave_probe = d_wp + w0; ra.wave_frame = d_wf + w0; ra.trans = d_tp;
                ra.nseg = nsegments; ra.seg = k; ra.slice = n; ra.nwaves = nw; ra.ny = g.ny; ra.hmax = ctx->hmax;
                ra.roots = ctx->d_roots_x;
                ra.tuples = d_tup + (size_t)tup_off[gi] * rpt; ra.ntuples = tup_off[gi + 1] - tup_off[gi];
                ra.pdl = step > 0;      // step 0 may directly follow the kernels that wrote t_n
                rc = launch_row(ctx, step == 0 ? ROW_FIRST : ROW_MID, ra, st);
                if (rc) return rc;
                const bool lastq = (step == total - 1) && output_space == 1;
                const bool fused = lastq && gt != nullptr;
                ColArgs ca{};
                ca.waves = ra.waves; ca.nwaves = nw; ca.nx = g.nx; ca.hmax = ctx->hmax; ca.roots = ctx->d_roots_y;
                ca.stack = (float2*)d_waves; ca.stack_waves = nwaves; ca.wave0 = w0;      // one tensor map for the whole call
                ca.px = ctx->d_px; ca.py = ctx->d_py; ca.kmax = ctx->d_kmax;
                // the tables carry 1/(nx ny): Psi_S unnormalised needs nx ny back; phi = Psi_S/sqrt(nx ny) needs sqrt(nx ny)
                ca.pscale = fused ? (float)std::sqrt((double)g.nx * (double)g.ny) : (lastq ? (float)((double)g.nx * (double)g.ny) : 1.f);
                ca.kmaxmax = ctx->kmaxmax;
                ca.pdl = 1;
                if (fused) { ca.roi_inv = gt->d_roi_inv; ca.wave_slot = d_ws + w0; ca.gbuf = gt->d_buf; ca.gq = gt->nroi; }
                rc = launch_col(ctx, fused ? COL_GATHER : (lastq ? COL_LASTQ : COL_MID), ca, g.ny, st);
                if (rc) return rc;
            }
        }
        if (output_space == 0) {
            RowArgs ra{};
            ra.waves = (float2*)d_waves + (size_t)w0 * npix; ra.nwaves = nw; ra.ny = g.ny; ra.hmax = ctx->hmax;
            ra.roots = ctx->d_roots_x;
            ra.pdl = 1;
            rc = launch_row(ctx, ROW_LAST, ra, st);
            if (rc) return rc;
        }
    }
    if (fork) {
        for (int i = 0; i + 1 < nstreams; ++i) {
            TACAW_CUDA(ctx, cudaEventRecord(ctx->ev_join[i], ctx->aux[i]));
            TACAW_CUDA(ctx, cudaStreamWaitEvent(user_st, ctx->ev_join[i], 0));
        }
    }
    return TACAW_OK;
}

int tacaw_propagate(tacaw_ctx* ctx, void* d_waves, const void* d_probes, int nprobes, const int32_t* wave_probe,
                    const int32_t* wave_frame, int nwaves, const void* const* d_trans, int nframes,
                    const int32_t* nslices_per_segment, int nsegments, double dz, int output_space, void* stream) {
    TACAW_ENTER(ctx);
    return propagate_impl(ctx, d_waves, d_probes, nprobes, wave_probe, wave_frame, nwaves, d_trans, nframes, nslices_per_segment,
                          nsegments, dz, output_space, nullptr, stream);
}

int tacaw_make_roi_inverse(tacaw_ctx* ctx, const int32_t* d_roi_idx, int64_t nroi, int32_t* d_roi_inv, void* stream) {
    TACAW_ENTER(ctx);
    if (nroi < 0 || !d_roi_inv || (nroi > 0 && !d_roi_idx)) return fail(ctx, TACAW_E_ARG, "tacaw_make_roi_inverse: bad argument");
    return launch_roi_inverse(ctx, d_roi_idx, nroi, d_roi_inv, (cudaStream_t)stream);
}

int tacaw_propagate_accumulate(tacaw_ctx* ctx, void* d_waves, const void* d_probes, int nprobes, const int32_t* wave_probe,
                               const int32_t* wave_frame, const int32_t* wave_time, int nwaves, const void* const* d_trans, int nframes,
                               const int32_t* nslices_per_segment, int nsegments, double dz, const int32_t* d_roi_inv, int64_t nroi,
                               void* d_buf, int nprobes_buf, int nframes_buf, void* stream) {
    TACAW_ENTER(ctx);
    if (nwaves < 0 || nroi < 0 || nprobes_buf <= 0 || nframes_buf <= 0 || (nwaves > 0 && (!wave_probe || !wave_time || !d_roi_inv || !d_buf)))
        return fail(ctx, TACAW_E_ARG, "tacaw_propagate_accumulate: bad argument");
    for (int w = 0; w < nwaves; ++w)
        if (wave_probe[w] < 0 || wave_probe[w] >= nprobes_buf || wave_time[w] < 0 || wave_time[w] >= nframes_buf)
            return fail(ctx, TACAW_E_ARG, "tacaw_propagate_accumulate: probe/frame index out of range");
    if (d_probes && nprobes > nprobes_buf) return fail(ctx, TACAW_E_ARG, "tacaw_propagate_accumulate: more probes than the buffer holds");
    GatherTarget gt{wave_time, d_roi_inv, nroi, (float2*)d_buf, nprobes_buf, nframes_buf};
    return propagate_impl(ctx, d_waves, d_probes, nprobes, wave_probe, wave_frame, nwaves, d_trans, nframes, nslices_per_segment,
                          nsegments, dz, 1, &gt, stream);
}

// O8 by row spans: for a fixed k every predicate is monotone in |h| (disc, annulus) or in h (rect), so the kept h of a row
// are one or two intervals whose ends are found by bisection on the fp64 predicate value; the cells are then emitted in
// ascending h.  (The oracle tests every cell; the two enumerators share the definition of theta^2 only.)
namespace {
struct RoiPred {
    const tacaw_grid* g;
    double lambda;
    bool square;
    double theta2(int h, int k) const {
        if (square) {
            const double sc = lambda / g->lx_A;
            return sc * sc * (double)((long long)h * h + (long long)k * k);
        }
        return lambda * lambda * ((h / g->lx_A) * (h / g->lx_A) + (k / g->ly_A) * (k / g->ly_A));
    }
};
// largest a in [0, amax] with theta2(a, k) <= lim2, or -1
int last_le(const RoiPred& p, int k, int amax, double lim2) {
    if (!(p.theta2(0, k) <= lim2)) return -1;
    int lo = 0, hi = amax + 1;
    while (hi - lo > 1) {
        const int mid = lo + (hi - lo) / 2;
        if (p.theta2(mid, k) <= lim2) lo = mid; else hi = mid;
    }
    return lo;
}
// smallest a in [0, amax] with theta2(a, k) >= lim2, or amax + 1
int first_ge(const RoiPred& p, int k, int amax, double lim2) {
    if (p.theta2(0, k) >= lim2) return 0;
    int lo = 0, hi = amax + 1;                       // theta2(lo) < lim2; hi: first candidate not yet excluded
    while (hi - lo > 1) {
        const int mid = lo + (hi - lo) / 2;
        if (p.theta2(mid, k) >= lim2) hi = mid; else lo = mid;
    }
    return hi;
}
}  // namespace

int tacaw_make_roi(const tacaw_grid* g, double lambda, int mode, const double* params, int32_t* idx_out, int64_t* count) {
    if (!g || !count || g->nx <= 0 || g->ny <= 0 || (mode != TACAW_ROI_FULL && !params)) return TACAW_E_ARG;
    if (mode < 0 || mode > 3) return TACAW_E_ARG;
    const RoiPred pred{g, lambda, g->nx == g->ny && g->lx_A == g->ly_A};
    const int hlo = -g->nx / 2, hhi = g->nx - g->nx / 2 - 1;        // signed h range of the grid
    const int amax = g->nx / 2;                                     // largest |h| (the negative end)
    int64_t c = 0;
    auto emit = [&](int k, int h0, int h1) {                        // cells h0..h1 of row k, clipped to the grid
        if (h0 < hlo) h0 = hlo;
        if (h1 > hhi) h1 = hhi;
        for (int h = h0; h <= h1; ++h, ++c)
            if (idx_out) idx_out[c] = (int32_t)(((k + g->ny) % g->ny) * g->nx + (h + g->nx) % g->nx);
    };
    for (int k = -g->ny / 2; k < g->ny - g->ny / 2; ++k) {
        if (mode == TACAW_ROI_FULL) {
            emit(k, hlo, hhi);
        } else if (mode == TACAW_ROI_DISC || mode == TACAW_ROI_ANNULUS) {
            const double to = (mode == TACAW_ROI_DISC) ? params[0] : params[1];
            const int aout = last_le(pred, k, amax, to * to);
            if (aout < 0) continue;
            int ain = 0;
            if (mode == TACAW_ROI_ANNULUS) ain = first_ge(pred, k, amax, params[0] * params[0]);
            if (ain > aout) continue;
            if (ain == 0) emit(k, -aout, aout);
            else { emit(k, -aout, -ain); emit(k, ain, aout); }
        } else {
            const double ty = lambda * k / g->ly_A;
            if (!(ty >= params[2] && ty <= params[3])) continue;
            // lambda*h/lx is increasing in h: first h with tx >= txmin, last h with tx <= txmax
            int lo = hlo - 1, hi = hhi + 1;
            while (hi - lo > 1) { const int mid = lo + (hi - lo) / 2; if (lambda * mid / g->lx_A >= params[0]) hi = mid; else lo = mid; }
            const int h0 = hi;
            lo = hlo - 1; hi = hhi + 1;
            while (hi - lo > 1) { const int mid = lo + (hi - lo) / 2; if (lambda * mid / g->lx_A <= params[1]) lo = mid; else hi = mid; }
            emit(k, h0, lo);
        }
    }
    *count = c;
    return TACAW_OK;
}

int tacaw_accumulate(tacaw_ctx* ctx, const void* d_qwaves, int nwaves, const int32_t* wave_probe,
                     const int32_t* wave_frame, const int32_t* d_roi_idx, int64_t nroi, void* d_buf, int nprobes,
                     int nframes, void* stream) {
    TACAW_ENTER(ctx);
    if (nwaves < 0 || nroi < 0 || nprobes <= 0 || nframes <= 0 ||
        (nwaves > 0 && nroi > 0 && (!d_qwaves || !wave_probe || !wave_frame || !d_roi_idx || !d_buf)))
        return fail(ctx, TACAW_E_ARG, "tacaw_accumulate: bad argument");
    if (nwaves == 0 || nroi == 0) return TACAW_OK;
    for (int w = 0; w < nwaves; ++w)
        if (wave_probe[w] < 0 || wave_probe[w] >= nprobes || wave_frame[w] < 0 || wave_frame[w] >= nframes)
            return fail(ctx, TACAW_E_ARG, "tacaw_accumulate: probe/frame index out of range");
    cudaStream_t st = (cudaStream_t)stream;
    // index arrays go to this entry point's own region (reuse is stream-ordered)
    size_t nb_i = sizeof(int) * (size_t)nwaves;
    void* reg = nullptr;
    int rc = region(ctx, tacaw_ctx::R_ACC, 2 * nb_i, &reg, "tacaw_accumulate");
    if (rc) return rc;
    int* d_wp = (int*)reg;
    int* d_wf = d_wp + nwaves;
    if ((rc = upload(ctx, d_wp, wave_probe, nb_i, st))) return rc;
    if ((rc = upload(ctx, d_wf, wave_frame, nb_i, st))) return rc;
    return launch_gather(ctx, (const float2*)d_qwaves, nwaves, d_wp, d_wf, d_roi_idx, nroi, (float2*)d_buf, nprobes,
                         nframes, st);
}

// Shared core of tacaw_spectrum / tacaw_spectrum_welch: chunks of L frames starting every `step` frames of a
// [nprobes][nframes_total][nroi] buffer, window table w[L] (fp64, host), I = (1/nchunks) sum_i I_i.
// chunk n starts at frame first + n*step and holds frames first + n*step + f*stride, f = 0..L-1; time step dt_fs (of a chunk).
static int spectrum_core(tacaw_ctx* ctx, const void* d_buf, int nprobes, int64_t nroi, int nframes_total, int L, int first, int step,
                         int stride, int nchunks, double dt_fs, const double* w, double temperature_K, double emin, double emax,
                         float* d_I, double* E_out, int* nE_out, cudaStream_t st, const char* who) {
    const bool pow2 = L >= 8 && L <= 2048 && (L & (L - 1)) == 0;
    if (!pow2 && (L < 2 || L > SPEC_DFT_MAX_L))
        return fail(ctx, TACAW_E_UNSUPPORTED, std::string(who) + ": the transform length must be a power of two in [8, 2048] or any length in [2, " +
                                                  std::to_string(SPEC_DFT_MAX_L) + "]");
    const double h_mev_fs = 4135.667696, kb_mev = 8.617333262e-2;
    // ascending axis k' = -L/2 .. L/2-1; keep [emin, emax] with 1e-9 meV slack (reading G11)
    int e_lo = -1, nE = 0;
    std::vector<double> E;
    // k' = -floor(L/2) .. L - floor(L/2) - 1 (for even L the Nyquist bin is the most negative energy)
    for (int i = 0; i < L; ++i) {
        double e = h_mev_fs * (double)(i - L / 2) / ((double)L * dt_fs);
        if (e < emin - 1e-9 || e > emax + 1e-9) continue;
        if (e_lo < 0) e_lo = i;
        E.push_back(e);
        ++nE;
    }
    *nE_out = nE;
    if (E_out) for (int i = 0; i < nE; ++i) E_out[i] = E[i];
    if (!d_I || nE == 0 || nprobes == 0 || nroi == 0 || nchunks == 0) return TACAW_OK;
    if (!d_buf) return fail(ctx, TACAW_E_ARG, std::string(who) + ": null buffer");
    if (!pow2) {
        // generic length: W[e][f] = w_f exp(-2 pi i k_e f/L) for the wanted bins only, then the per-energy factor
        double sw2g = 0.0;
        for (int f = 0; f < L; ++f) sw2g += w[f] * w[f];
        if (!(sw2g > 0)) return fail(ctx, TACAW_E_ARG, std::string(who) + ": window is identically zero");
        std::vector<float> tabg(2 * (size_t)nE * L + (size_t)nE);
        for (int i = 0; i < nE; ++i) {
            const long long kp = (long long)(e_lo + i) - L / 2;           // signed bin
            for (int f = 0; f < L; ++f) {
                const long long m = (((kp * f) % L) + L) % L;
                const double ang = -2.0 * M_PI * (double)m / (double)L;
                tabg[2 * ((size_t)i * L + f)] = (float)(w[f] * std::cos(ang));
                tabg[2 * ((size_t)i * L + f) + 1] = (float)(w[f] * std::sin(ang));
            }
            const double x = E[i] / (kb_mev * temperature_K);
            const double B = (x == 0.0) ? 1.0 : x / (-std::expm1(-x));
            tabg[2 * (size_t)nE * L + i] = (float)(B / ((double)L * sw2g * (double)nchunks));
        }
        void* regg = nullptr;
        int rcg = region(ctx, tacaw_ctx::R_SPEC, sizeof(float) * tabg.size(), &regg, who);
        if (rcg) return rcg;
        if ((rcg = upload(ctx, regg, tabg.data(), sizeof(float) * tabg.size(), st))) return rcg;
        return launch_spectrum_dft(ctx, (const float2*)d_buf + (size_t)first * (size_t)nroi, nprobes, nroi, L,
                                   (size_t)nframes_total * (size_t)nroi, (size_t)stride * (size_t)nroi, nchunks, (size_t)step * (size_t)nroi,
                                   (const float2*)regg, (const float*)regg + 2 * (size_t)nE * L, nE, d_I, st);
    }
    // table region: roots exp(-2 pi i j/L) (L < 512) or the single-exchange twiddle table of fft2.cuh (L >= 512); window; bose
    static const bool two_exchange = [] { const char* e = getenv("TACAW_SPEC_TWO_EXCHANGE"); return e && atoi(e) != 0; }();
    const bool plan2 = L >= 512 && !two_exchange;
    const size_t ntw = plan2 ? (size_t)fft2_table_elems(L) : (size_t)L;
    const size_t NR = ntw > (size_t)L ? ntw : (size_t)L;               // float2 entries reserved for the table
    std::vector<float> tab(2 * NR + (size_t)L + (size_t)nE);
    double sw2 = 0.0;
    for (int f = 0; f < L; ++f) sw2 += w[f] * w[f];
    if (!(sw2 > 0)) return fail(ctx, TACAW_E_ARG, std::string(who) + ": window is identically zero");
    if (plan2) fft2_host_table(L, reinterpret_cast<float2*>(tab.data()));
    for (int j = 0; j < L; ++j) {
        if (!plan2) {
            double ang = -2.0 * M_PI * (double)j / (double)L;
            tab[2 * j] = (float)std::cos(ang);
            tab[2 * j + 1] = (float)std::sin(ang);
        }
        tab[2 * NR + j] = (float)w[j];
    }
    for (int i = 0; i < nE; ++i) {
        double x = E[i] / (kb_mev * temperature_K);
        double B = (x == 0.0) ? 1.0 : x / (-std::expm1(-x));
        tab[2 * NR + (size_t)L + i] = (float)(B / ((double)L * sw2 * (double)nchunks));
    }
    void* reg = nullptr;
    int rc = region(ctx, tacaw_ctx::R_SPEC, sizeof(float) * tab.size(), &reg, who);
    if (rc) return rc;
    float* d_spec_tab = (float*)reg;
    if ((rc = upload(ctx, d_spec_tab, tab.data(), sizeof(float) * tab.size(), st))) return rc;
    // one launch for all chunks: the kernel sums |Phi_n|^2 over the chunks in registers and writes I once
    return launch_spectrum(ctx, (const float2*)d_buf + (size_t)first * (size_t)nroi, nprobes, nroi, L,
                           (size_t)nframes_total * (size_t)nroi, (size_t)stride * (size_t)nroi, nchunks, (size_t)step * (size_t)nroi,
                           (const float2*)d_spec_tab, d_spec_tab + 2 * NR, d_spec_tab + 2 * NR + (size_t)L, e_lo, nE, d_I, st);
}

// modified Bessel function I0 (power series; converges for every beta used as a Kaiser parameter)
static double bessel_i0(double x) {
    double sum = 1.0, term = 1.0;
    const double q = 0.25 * x * x;
    for (int k = 1; k < 500; ++k) {
        term *= q / ((double)k * (double)k);
        sum += term;
        if (term < 1e-17 * sum) break;
    }
    return sum;
}

// Dolph-Chebyshev: periodic form of the M = n + 1 point window whose transform is T_{M-1}(x0 cos(theta/2)):
// cosine series over the M samples of that transform, centred on the window's midpoint, angles reduced in integer
// arithmetic before cos(), normalised to its maximum.
static int dolph_chebyshev(int n, double att_db, double* w_out) {
    if (!(att_db > 0.0)) return TACAW_E_ARG;
    const int M = n + 1, m = M - 1;
    const double x0 = std::cosh(std::acosh(std::pow(10.0, att_db / 20.0)) / (double)m);
    std::vector<double> Wk(M);
    for (int k = 0; k < M; ++k) {
        const double x = x0 * std::cos(M_PI * (double)k / (double)M);
        double t;
        if (x > 1.0) t = std::cosh((double)m * std::acosh(x));
        else if (x < -1.0) t = ((m & 1) ? -1.0 : 1.0) * std::cosh((double)m * std::acosh(-x));
        else t = std::cos((double)m * std::acos(x));
        Wk[k] = t;
    }
    std::vector<double> w(M);
    double wmax = 0.0;
    for (int j = 0; j < M; ++j) {
        double acc = Wk[0];
        for (int k = 1; k < M; ++k) {
            // reduce the angle 2 pi k d / M through the integer 2 k j - k m (mod 2M) before calling cos
            const long long num = ((2LL * k * j - (long long)k * m) % (2LL * M) + 2LL * M) % (2LL * M);
            acc += Wk[k] * std::cos(M_PI * (double)num / (double)M);
        }
        w[j] = acc;
        if (acc > wmax) wmax = acc;
    }
    for (int f = 0; f < n; ++f) w_out[f] = w[f] / wmax;
    return TACAW_OK;
}

int tacaw_make_window(int kind, int n, double param, double* w_out) {
    if (n <= 0 || !w_out) return TACAW_E_ARG;
    if (kind == TACAW_WINDOW_DOLPH_CHEBYSHEV) return dolph_chebyshev(n, param, w_out);
    for (int f = 0; f < n; ++f) {
        const double x = (double)f / (double)n;          // periodic form: sample f of a window of period n
        double v = 1.0;
        switch (kind) {
            case TACAW_WINDOW_RECT: v = 1.0; break;
            case TACAW_WINDOW_HANN: v = 0.5 - 0.5 * std::cos(2.0 * M_PI * x); break;
            case TACAW_WINDOW_TUKEY: {
                const double a = param;
                if (!(a >= 0.0 && a <= 1.0)) return TACAW_E_ARG;
                if (a == 0.0) v = 1.0;
                else if (x < 0.5 * a) v = 0.5 * (1.0 - std::cos(2.0 * M_PI * x / a));
                else if (x <= 1.0 - 0.5 * a) v = 1.0;
                else v = 0.5 * (1.0 - std::cos(2.0 * M_PI * (1.0 - x) / a));
                break;
            }
            case TACAW_WINDOW_BLACKMAN_HARRIS:
                v = 0.35875 - 0.48829 * std::cos(2.0 * M_PI * x) + 0.14128 * std::cos(4.0 * M_PI * x) - 0.01168 * std::cos(6.0 * M_PI * x);
                break;
            case TACAW_WINDOW_KAISER: {
                if (!(param >= 0.0)) return TACAW_E_ARG;
                const double u = 2.0 * x - 1.0;
                v = bessel_i0(param * std::sqrt(std::fmax(0.0, 1.0 - u * u))) / bessel_i0(param);
                break;
            }
            default: return TACAW_E_ARG;
        }
        w_out[f] = v;
    }
    return TACAW_OK;
}

int tacaw_spectrum(tacaw_ctx* ctx, const void* d_buf, int nprobes, int64_t nroi, int nframes, double dt_fs, int window,
                   double temperature_K, double emin, double emax, float* d_I, double* E_out, int* nE_out, void* stream) {
    TACAW_ENTER(ctx);
    if (nprobes < 0 || nroi < 0 || nframes <= 0 || !(dt_fs > 0) || !(temperature_K > 0) || !nE_out ||
        (window != TACAW_WINDOW_RECT && window != TACAW_WINDOW_HANN))
        return fail(ctx, TACAW_E_ARG, "tacaw_spectrum: bad argument");
    std::vector<double> w(nframes);
    tacaw_make_window(window, nframes, 0.0, w.data());
    return spectrum_core(ctx, d_buf, nprobes, nroi, nframes, nframes, 0, nframes, 1, 1, dt_fs, w.data(), temperature_K, emin, emax, d_I,
                         E_out, nE_out, (cudaStream_t)stream, "tacaw_spectrum");
}

int tacaw_spectrum_welch(tacaw_ctx* ctx, const void* d_buf, int nprobes, int64_t nroi, int nframes_total, int chunk_len,
                         int chunk_overlap, int skip_init, int frame_stride, double dt_fs, const double* window_table,
                         double temperature_K, double emin, double emax, float* d_I, double* E_out, int* nE_out, int* nchunks_out,
                         void* stream) {
    TACAW_ENTER(ctx);
    if (nprobes < 0 || nroi < 0 || nframes_total <= 0 || chunk_len <= 0 || chunk_overlap <= 0 || skip_init < 0 || frame_stride <= 0 ||
        !(dt_fs > 0) || !(temperature_K > 0) || !nE_out || !window_table)
        return fail(ctx, TACAW_E_ARG, "tacaw_spectrum_welch: bad argument");
    // s_{n+1} = s_n + L/nu, remainder-less division, counted in the chunk's own snapshots: with a stride the
    // next chunk starts (L/nu)*stride stored frames later (reading G24)
    const long long step = (long long)(chunk_len / chunk_overlap) * frame_stride;
    if (step <= 0) return fail(ctx, TACAW_E_ARG, "tacaw_spectrum_welch: chunk_overlap exceeds chunk_len");
    const long long span = (long long)(chunk_len - 1) * frame_stride + 1;      // stored frames a chunk covers
    int nchunks = 0;
    for (long long s0 = skip_init; s0 + span <= nframes_total; s0 += step) ++nchunks;
    if (nchunks_out) *nchunks_out = nchunks;
    return spectrum_core(ctx, d_buf, nprobes, nroi, nframes_total, chunk_len, skip_init, (int)step, frame_stride, nchunks,
                         dt_fs * frame_stride, window_table, temperature_K, emin, emax, d_I, E_out, nE_out, (cudaStream_t)stream,
                         "tacaw_spectrum_welch");
}

int tacaw_make_scan(int mode, const int32_t* shape, const double* origin, const double* a, const double* b, const double* cell,
                    double* xy_out) {
    if (!shape || !origin || !a || !xy_out || shape[0] <= 0 || shape[1] <= 0) return TACAW_E_ARG;
    if (mode < TACAW_SCAN_BOX || mode > TACAW_SCAN_PARALLELOGRAM) return TACAW_E_ARG;
    if ((mode == TACAW_SCAN_PARALLELOGRAM && !b) || (mode == TACAW_SCAN_BOX_RELATIVE && !cell)) return TACAW_E_ARG;
    const int n0 = shape[0], n1 = shape[1];
    // edge vectors e0 (along i) and e1 (along j) and the start corner, in Angstrom; end point excluded (:380)
    double o[2] = {origin[0], origin[1]}, e0[2] = {0.0, 0.0}, e1[2] = {0.0, 0.0};
    switch (mode) {
        case TACAW_SCAN_BOX: e0[0] = a[0] - origin[0]; e1[1] = a[1] - origin[1]; break;
        case TACAW_SCAN_UNITCELL: e0[0] = a[0]; e1[1] = a[1]; break;
        case TACAW_SCAN_PARALLELOGRAM: e0[0] = a[0]; e0[1] = a[1]; e1[0] = b[0]; e1[1] = b[1]; break;
        default: break;
    }
    for (int i = 0; i < n0; ++i)
        for (int j = 0; j < n1; ++j) {
            const double fi = (double)i / (double)n0, fj = (double)j / (double)n1;
            double* r = xy_out + 2 * ((size_t)i * n1 + j);
            if (mode == TACAW_SCAN_BOX_RELATIVE) {
                r[0] = (origin[0] + fi * (a[0] - origin[0])) * cell[0];
                r[1] = (origin[1] + fj * (a[1] - origin[1])) * cell[1];
            } else {
                r[0] = o[0] + fi * e0[0] + fj * e1[0];
                r[1] = o[1] + fi * e0[1] + fj * e1[1];
            }
        }
    return TACAW_OK;
}

int tacaw_scan_batch(const int32_t* shape, const int32_t* bs, int batch, int32_t* idx_out, int32_t* count, int32_t* nbatches) {
    if (!shape || !bs || !count || shape[0] <= 0 || shape[1] <= 0 || bs[0] <= 0 || bs[1] <= 0) return TACAW_E_ARG;
    const int t0 = (shape[0] + bs[0] - 1) / bs[0], t1 = (shape[1] + bs[1] - 1) / bs[1];
    if (nbatches) *nbatches = t0 * t1;
    if (batch < 0 || batch >= t0 * t1) return TACAW_E_ARG;
    const int i0 = (batch / t1) * bs[0], j0 = (batch % t1) * bs[1];
    const int i1 = i0 + bs[0] < shape[0] ? i0 + bs[0] : shape[0], j1 = j0 + bs[1] < shape[1] ? j0 + bs[1] : shape[1];
    int32_t c = 0;
    for (int i = i0; i < i1; ++i)
        for (int j = j0; j < j1; ++j, ++c)
            if (idx_out) idx_out[c] = i * shape[1] + j;
    *count = c;
    return TACAW_OK;
}

int tacaw_make_detector(const tacaw_grid* g, double lambda, int kind, const double* center, const double* radii,
                        const int32_t* roi_idx, int64_t nroi, float* w_out) {
    if (!g || g->nx <= 0 || g->ny <= 0 || !center || !radii || nroi < 0 || (nroi > 0 && (!roi_idx || !w_out))) return TACAW_E_ARG;
    if (kind != TACAW_DETECTOR_CIRCULAR && kind != TACAW_DETECTOR_ANNULAR) return TACAW_E_ARG;
    if (!(radii[1] >= 0) || (kind == TACAW_DETECTOR_ANNULAR && !(radii[0] >= 0 && radii[0] <= radii[1]))) return TACAW_E_ARG;
    const long long npix = (long long)g->nx * g->ny;
    for (int64_t r = 0; r < nroi; ++r) {
        const long long idx = roi_idx[r];
        if (idx < 0 || idx >= npix) return TACAW_E_ARG;
        const int h = sgn_index((int)(idx % g->nx), g->nx), k = sgn_index((int)(idx / g->nx), g->ny);
        const double tx = lambda * h / g->lx_A - center[0], ty = lambda * k / g->ly_A - center[1];
        const double t2 = tx * tx + ty * ty;
        bool on = t2 <= radii[1] * radii[1];
        if (kind == TACAW_DETECTOR_ANNULAR) on = on && t2 >= radii[0] * radii[0];
        w_out[r] = on ? 1.0f : 0.0f;
    }
    return TACAW_OK;
}

int tacaw_detect(tacaw_ctx* ctx, const float* d_I, int nprobes, int nE, int64_t nroi, const float* d_weights, int ndet,
                 float* d_out, void* stream) {
    TACAW_ENTER(ctx);
    if (nprobes < 0 || nE < 0 || nroi < 0 || ndet <= 0 || ((nprobes > 0 && nE > 0) && (!d_out || (nroi > 0 && (!d_I || !d_weights)))))
        return fail(ctx, TACAW_E_ARG, "tacaw_detect: bad argument");
    return launch_detect(ctx, d_I, nprobes, nE, nroi, d_weights, ndet, d_out, (cudaStream_t)stream);
}

}  // extern "C"

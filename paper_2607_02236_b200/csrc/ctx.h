// ctx.h -- internal context of libtacaw (not part of the ABI).
#pragma once
#include <cuda_runtime.h>

#include <cuda.h>

#include <cstdint>
#include <string>
#include <unordered_map>
#include <vector>

#include "../../include/tacaw.h"

struct tacaw_ctx {
    tacaw_grid grid{};
    tacaw_beam beam{};
    int device = 0;
    int num_sms = 148;
    size_t l2_bytes = 0;

    float2* d_roots_x = nullptr;  // twiddle table of the length-nx transforms (fft2.cuh layout)
    float2* d_roots_y = nullptr;  // same for length ny
    int* d_kmax = nullptr;        // [nx] per column ix: largest |k| inside the band-limit mask, -1 = none
    int* d_kmax_pot = nullptr;    // [nx] same for the potential (Nyquist row/column excluded)
    std::vector<int> kmax, kmax_pot;
    int hmax = 0;                 // largest |h| with any in-band k  (propagator mask)
    int hmax_pot = 0;             // same for the potential
    int kmaxmax_pot = 0;
    int kmaxmax = 0;              // largest kmax[ix]

    bool generic_path = false;    // nx or ny is not a power of two: both passes run on generic.cu (tables = plain roots of unity)

    double dz_cached = -1.0;
    float2* d_px = nullptr;  // [nx] exp(-i pi lambda dz h^2/lx^2) / nx
    float2* d_py = nullptr;  // [ny] exp(-i pi lambda dz k^2/ly^2) / ny

    // Workspace: ONE caller-owned device buffer (tacaw_set_workspace), cut into one region per entry point so that
    // no two entry points share scratch.  The library never allocates device memory after tacaw_create.
    enum Region { R_BUILD = 0, R_STAGE, R_PROBE, R_PROP, R_ACC, R_SPEC, R_COUNT };
    char* d_ws = nullptr;
    size_t ws_bytes = 0;
    size_t reg_off[R_COUNT] = {0}, reg_bytes[R_COUNT] = {0};
    int* d_flags = nullptr;       // [4] sticky device-side error flags ([0]: species id out of range), owned by the context

    // pinned host arena for per-call index arrays: lets cudaMemcpyAsync return without draining
    // the stream (a pageable source would synchronise it).  Two halves, each guarded by an event recorded
    // after the last copy issued from it, so reuse waits for exactly those copies.
    char* h_arena = nullptr;
    size_t arena_bytes = 0, arena_off = 0;
    cudaEvent_t ev_arena[2] = {nullptr, nullptr};
    bool arena_used[2] = {false, false};

    // per-context (= per-device) kernel state: opt-in shared-memory attribute set / occupancy of each kernel
    std::unordered_map<const void*, int> kernel_occ;
    // tensor maps of wave stacks already encoded (key: base pointer, rows, box)
    struct MapEntry { const void* base; long long rows; int nx, box_cols, box_rows; alignas(64) CUtensorMap tm; };
    std::vector<MapEntry> maps;

    // internal streams: tacaw_propagate runs wave groups round-robin on the caller's stream and these, so one group's
    // kernel tails overlap the other groups' kernels (fork/join with events around the call; TACAW_STREAMS, default 3)
    static constexpr int MAX_AUX = 3;
    cudaStream_t aux[MAX_AUX] = {nullptr, nullptr, nullptr};
    cudaEvent_t ev_fork = nullptr, ev_join[MAX_AUX] = {nullptr, nullptr, nullptr};

    std::string err;
    int64_t launches = 0;
};

namespace tacaw {

int fail(tacaw_ctx* ctx, int code, const std::string& msg);
int cuda_fail(tacaw_ctx* ctx, cudaError_t e, const char* where);
// region `r` of the caller's workspace if it holds `need` bytes, else TACAW_E_NOMEM (no allocation ever happens here)
int region(tacaw_ctx* ctx, int r, size_t need, void** out, const char* who);
// makes ctx->device current for the lifetime of the object and restores the caller's device afterwards
struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(const tacaw_ctx* ctx) {
        if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; ok = false; return; }
        if (prev != ctx->device && cudaSetDevice(ctx->device) != cudaSuccess) ok = false;
    }
    ~DeviceGuard() {
        int cur = -1;
        if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev);
    }
};
#define TACAW_ENTER(ctx)                                                   \
    if (!(ctx)) return TACAW_E_ARG;                                        \
    tacaw::DeviceGuard guard__(ctx);                                       \
    if (!guard__.ok) return tacaw::fail(ctx, TACAW_E_CUDA, "cannot make the context's device current")
// async H2D of a small host array through the pinned arena (falls back to a pageable copy)
int upload(tacaw_ctx* ctx, void* dst, const void* src, size_t bytes, cudaStream_t st);

constexpr int MAX_SPECIES = 8;
struct AbTable {
    float a[MAX_SPECIES][4];
    float b[MAX_SPECIES][4];
};

#define TACAW_CUDA(ctx, call)                                        \
    do {                                                             \
        cudaError_t e__ = (call);                                    \
        if (e__ != cudaSuccess) return tacaw::cuda_fail(ctx, e__, #call); \
    } while (0)

// launchers implemented in the kernel translation units --------------------------------------
enum RowMode { ROW_FIRST = 0, ROW_MID = 1, ROW_LAST = 2, ROW_TRANS = 3 };
enum ColMode { COL_MID = 0, COL_LASTQ = 1, COL_INV = 2, COL_GATHER = 3 };

struct RowArgs {
    float2* waves;                 // [nwaves][ny][nx]
    const float2* probes;          // or nullptr
    const int* wave_probe;         // device
    const int* wave_frame;         // device
    const float2* const* trans;    // device [nframes*nseg] segment base pointers
    int nseg, seg, slice;          // which t_n this step uses: trans[f*nseg+seg] + slice*ny*nx
    int nwaves, ny;
    const int* tuples;             // device [ntuples][rows per team] wave indices (same frame within a tuple), or
    int ntuples;                   //   nullptr: tuple p = waves p*RPT .. (set by the launcher)
    int pdl;                       // launch as a programmatic dependent of the previous kernel in the stream
    int hmax;                      // in-band columns: ix <= hmax || ix >= nx-hmax
    long long nitems;              // (row, tuple) work items; set by the launcher
    int ipc;                       // items per CTA; set by the launcher
    const float2* roots;           // twiddle table of length-nx transforms
    float scale;                   // ROW_TRANS: sigma/(lx ly)
};

struct ColArgs {
    float2* waves;                 // first wave of this launch
    float2* stack;                 // the wave stack the tensor map describes (nullptr: `waves` itself) ...
    int stack_waves, wave0;        //   ... its length and the index of waves[0] in it
    int nwaves, nx;
    int hmax;
    long long nitems;              // (column group, wave) work items; set by the launcher
    int ipc;                       // items per CTA; set by the launcher
    const float2* roots;           // twiddle table of length-ny transforms
    const float2* px;
    const float2* py;
    const int* kmax;
    float pscale;                  // multiplies px*py (1 for COL_MID, nx*ny for COL_LASTQ)
    int pdl;                       // launch as a programmatic dependent of the previous kernel in the stream
    int kmaxmax;                   // largest kmax[ix] of the masked modes (-1: not applicable)
    // COL_GATHER (fused a6): the ROI pixels of Psi_S go straight into the time-ordered buffer
    const int* roi_inv;            // device [ny][nx]: ROI position r of a pixel, -1 outside the ROI
    const int* wave_slot;          // device [nwaves]: probe * nframes_buf + frame of each wave of this launch
    float2* gbuf;                  // buffer [nprobes][nframes][nroi]
    long long gq;                  // nroi
};

int launch_row(tacaw_ctx* ctx, int mode, const RowArgs& a, cudaStream_t st);
int row_tuple_size(int nx);        // waves per tuple of the row kernel for this grid width
int slice_step_table_elems(int n); // twiddle table of the slice-step transforms of length n (fft2.cuh XPlan layout) ...
void slice_step_host_table(int n, float2* tab);   // ... built on the host in fp64
int launch_col(tacaw_ctx* ctx, int mode, const ColArgs& a, int ny, cudaStream_t st);
// grids that are not powers of two (generic.cu): even n <= 2048 with prime factors 2, 3, 5, 7 (the paper's 1680)
bool generic_grid_supported(int n);
int launch_row_generic(tacaw_ctx* ctx, int mode, const RowArgs& a, cudaStream_t st);
int launch_col_generic(tacaw_ctx* ctx, int mode, const ColArgs& a, int ny, cudaStream_t st);
void generic_host_table(int n, float2* tab);      // n roots of unity exp(-2 pi i m / n)

// d_nclamped (out): device address of this call's clamp counter inside the build region
int launch_potential(tacaw_ctx* ctx, const double* d_pos, const int32_t* d_species, int natoms, int nframes, int nspecies,
                     const AbTable& ab, double dz, int nslices, double z0, float2* d_V, int** d_nclamped,
                     cudaStream_t st);
// the same with the build region in a static device array of TACAW_STATIC_SCRATCH_BYTES (potential.cu); no workspace needed
int launch_potential_static(tacaw_ctx* ctx, const double* d_pos, const int32_t* d_species, int natoms, int nframes, int nspecies,
                            const AbTable& ab, double dz, int nslices, double z0, float2* d_V, cudaStream_t st);
// tensor-core K1 (potential_tc.cu): sorted fixed-point coordinates and per-(slice, species) offsets -> V(q) of every slice
int launch_potential_tc(tacaw_ctx* ctx, const uint32_t* sx, const uint32_t* sy, const int* offsets, int nspecies, const AbTable& ab,
                        int nslices_total, float2* d_V, cudaStream_t st);
int potential_tc_max_species();
// series of a length that is not a power of two (<= SPEC_DFT_MAX_L): plain DFT restricted to the nE wanted bins, W [nE][L]
int launch_spectrum_dft(tacaw_ctx* ctx, const float2* d_buf, int nprobes, int64_t nroi, int L, size_t probe_stride, size_t frame_stride,
                        int nchunks, size_t chunk_stride, const float2* d_W, const float* d_bose, int nE, float* d_I, cudaStream_t st);
constexpr int SPEC_DFT_MAX_L = 512;
// spectrum region: twiddle/window/Bose tables of one call, or the [nE][L] DFT table of the generic path
constexpr size_t SPEC_TABLE_BYTES = (size_t)SPEC_DFT_MAX_L * SPEC_DFT_MAX_L * 8 + 16 * 1024;
int launch_probe_fill(tacaw_ctx* ctx, const uint32_t* d_uxy /*[P][2] fixed-point fractional*/, int nprobes,
                      const int* d_kap /*[nx]*/, float amp, float2* d_waves, cudaStream_t st);
int launch_roi_inverse(tacaw_ctx* ctx, const int* d_idx, int64_t nroi, int* d_inv, cudaStream_t st);
int launch_zero_slots(tacaw_ctx* ctx, float2* d_buf, const int* d_slot, int nwaves, int64_t nroi, cudaStream_t st);
int launch_gather(tacaw_ctx* ctx, const float2* d_q, int nwaves, const int* d_wp, const int* d_wf, const int* d_idx,
                  int64_t nroi, float2* d_buf, int nprobes, int nframes, cudaStream_t st);
// probe_stride / frame_stride / chunk_stride: elements between consecutive probes' series blocks, consecutive frames of a
// chunk, and the first frames of consecutive Welch chunks; all nchunks chunks are transformed and summed in one launch
int launch_spectrum(tacaw_ctx* ctx, const float2* d_buf, int nprobes, int64_t nroi, int nframes, size_t probe_stride,
                    size_t frame_stride, int nchunks, size_t chunk_stride, const float2* d_roots,
                    const float* d_window, const float* d_bose, int e_lo, int nE, float* d_I, cudaStream_t st);

int launch_detect(tacaw_ctx* ctx, const float* d_I, int nprobes, int nE, int64_t nroi, const float* d_w, int ndet, float* d_out,
                  cudaStream_t st);

}  // namespace tacaw

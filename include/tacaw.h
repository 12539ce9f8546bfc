/* tacaw.h -- C ABI of the B200-native TACAW hot path (libtacaw.so, hand-written sm_100a CUDA).
 *
 * Method: arxiv/paper_2607_02236 ("torched-TACAW").  Citations are PAPER.md line numbers.
 *   I(q,E) ~ beta E/(1-exp(-beta E)) |phi_MD(q,E)|^2                      Eq.(1), :35-40
 *   one batch = multislice on each snapshot, gather of the exit wave inside a q-ROI, window,
 *   time->energy FFT, |.|^2, quantum-statistics factor                      :122, :132, :142
 * The multislice formulas (the paper delegates them to pyms, :94) are the textbook scheme that
 * DESIGN.md section 3 spells out (steps O1-O10, readings G1-G21).
 *
 * Conventions
 *   - Arrays are row-major [iy][ix], x fastest.  complex64 = interleaved (re, im) float.
 *   - Frequency index h = ix for ix < nx/2, else ix - nx (same for k, iy).  q = (h/lx, k/ly) in
 *     1/Angstrom (no 2 pi).  Forward transform uses exp(-2 pi i ...); inverse carries 1/(nx ny).
 *   - nx, ny in [16, 2048] (they may differ): powers of two run on the register FFTs of the tuned kernels; any other EVEN
 *     size whose prime factors are 2, 3, 5, 7 only (the paper's 1680 = 2^4 3 5 7) runs on a plain mixed-radix
 *     path (same results and tolerances, several times slower).  Anything else: TACAW_E_UNSUPPORTED.
 *   - Every "d_" pointer is DEVICE memory owned by the caller; the library never frees or
 *     reallocates it.  The library owns only the context (twiddle / propagator tables, a pinned host
 *     arena for index uploads, streams and events) -- all created in tacaw_create.  Scratch for the
 *     calls is ONE caller-owned device buffer (tacaw_workspace_bytes / tacaw_set_workspace): no call
 *     allocates, frees or device-synchronises.  A call whose scratch does not fit returns TACAW_E_NOMEM.
 *   - `stream` is a cudaStream_t cast to void* (NULL = default stream).  Calls enqueue work on it
 *     and return without synchronising unless stated; host outputs are written before return.
 *   - ONE STREAM AT A TIME PER CONTEXT: consecutive calls on a context must be issued on the same stream, or be
 *     ordered by the caller (event / synchronise) when the stream changes -- the workspace regions and the
 *     propagator tables are reused in stream order.  To overlap, e.g., tacaw_build_slices of the next frame block
 *     with tacaw_propagate of the current one, use two contexts (each with its own workspace).
 *   - Every entry point makes the context's device current for the duration of the call and restores the caller's
 *     current device before returning.
 *   - Every call returns TACAW_OK (0) or a negative TACAW_E_* code; nothing throws or exits.
 *     tacaw_last_error(ctx) gives a message for the last failure on that context.
 *   - There is no CPU fallback: without a CUDA device tacaw_create fails with TACAW_E_CUDA.
 */
#ifndef TACAW_H
#define TACAW_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TACAW_OK 0
#define TACAW_E_ARG (-1)         /* bad argument (null pointer, negative size, index out of range) */
#define TACAW_E_UNSUPPORTED (-2) /* grid or series length outside the supported set */
#define TACAW_E_NOMEM (-3)       /* the caller's workspace is missing or too small for this call */
#define TACAW_E_CUDA (-4)        /* CUDA runtime error (message in tacaw_last_error) */

typedef struct tacaw_ctx tacaw_ctx;

typedef struct {
    int nx, ny;       /* grid points */
    double lx_A, ly_A; /* periodic cell edge lengths, Angstrom */
} tacaw_grid;

typedef struct {
    double lambda_A;          /* electron wavelength, Angstrom */
    double sigma_rad_per_VA;  /* interaction constant, rad/(V Angstrom) */
    int bandlimit;            /* 1: sharp mask at 2/3 of the smaller Nyquist (O5, reading G3); 0: none */
} tacaw_beam;

typedef struct {
    int nspecies;
    const double *a; /* HOST [nspecies][4], V*Angstrom^3 */
    const double *b; /* HOST [nspecies][4], Angstrom^2   : f_s(q^2) = sum_i a_si exp(-b_si q^2) */
} tacaw_species;

/* ROI predicates for tacaw_make_roi (O8). */
#define TACAW_ROI_FULL 0
#define TACAW_ROI_DISC 1     /* params: theta_o                    lambda^2 q^2 <= theta_o^2       */
#define TACAW_ROI_ANNULUS 2  /* params: theta_i, theta_o                                            */
#define TACAW_ROI_RECT 3     /* params: txmin, txmax, tymin, tymax  (the paper's minmax_mrad), rad  */

#define TACAW_WINDOW_RECT 0
#define TACAW_WINDOW_HANN 1  /* periodic Hann, w_f = 1/2 - 1/2 cos(2 pi f/T) (:142, :182; reading G9) */
/* further windows of tacaw_make_window (Appendix A), all in the periodic form x = f/n */
#define TACAW_WINDOW_TUKEY 2            /* param = alpha in [0,1]: cosine tapers of total fractional width alpha; 1 = Hann, 0 = rect (:170) */
#define TACAW_WINDOW_BLACKMAN_HARRIS 3  /* 4-term, 0.35875 - 0.48829 cos(2 pi x) + 0.14128 cos(4 pi x) - 0.01168 cos(6 pi x) */
#define TACAW_WINDOW_KAISER 4           /* param = beta >= 0: I0(beta sqrt(1 - (2x-1)^2)) / I0(beta) */
#define TACAW_WINDOW_DOLPH_CHEBYSHEV 5  /* param = side-lobe attenuation in dB > 0 (the paper uses 100 dB, :352): the window whose
                                           transform is the Chebyshev polynomial T_n(x0 cos(theta/2)), x0 = cosh(acosh(10^(dB/20))/n),
                                           i.e. every side lobe `param` dB below the main lobe; max = 1 */

/* Library version string and the SM architecture it was compiled for ("sm_100a"). */
const char *tacaw_version(void);

/* Create a context on CUDA device `device`: twiddle tables, band-limit column extents.
 * Fails with TACAW_E_UNSUPPORTED for grids outside the supported set, TACAW_E_CUDA without a GPU. */
int tacaw_create(tacaw_ctx **ctx, const tacaw_grid *grid, const tacaw_beam *beam, int device);
int tacaw_destroy(tacaw_ctx *ctx);
const char *tacaw_last_error(const tacaw_ctx *ctx);

/* Workspace ("every device buffer is allocated by the caller").  tacaw_sizes announces the LARGEST
 * call of each kind the caller will make; tacaw_workspace_bytes returns the bytes those calls need in total (each entry
 * point gets its own 256-byte aligned region, so no two entry points share scratch); tacaw_set_workspace hands the
 * library a device buffer of at least that size (256-byte aligned; it stays the caller's and must outlive every call
 * queued against it).  It may be called again with a larger buffer once the work queued on the old one is ordered
 * before the next call (same stream).  Calls that need no scratch (tacaw_detect, the HOST helpers) work without one. */
typedef struct {
    int natoms;       /* atoms per tacaw_build_slices call (one z-segment) */
    int nframes;      /* frames per tacaw_build_slices call and frames in flight per tacaw_propagate call */
    int nslices;      /* slices per tacaw_build_slices call (largest segment) */
    int nsegments;    /* z-segments per tacaw_propagate call (0 = 1) */
    int nwaves;       /* waves per tacaw_propagate / tacaw_accumulate call */
    int nprobes;      /* probes per tacaw_make_probes call */
    int host_staging; /* 1: also reserve the staging region of tacaw_build_slices_host (natoms x nframes positions) */
} tacaw_sizes;
size_t tacaw_workspace_bytes(const tacaw_ctx *ctx, const tacaw_sizes *sizes);
int tacaw_set_workspace(tacaw_ctx *ctx, void *d_workspace, size_t bytes, const tacaw_sizes *sizes);

/* Device-side error flags raised by kernels since the last check (at present: a species id outside
 * [0, nspecies) seen by tacaw_build_slices, which then uses species 0 for that atom).  Synchronises `stream`,
 * returns TACAW_E_ARG and clears the flags if any was raised, TACAW_OK otherwise. */
int tacaw_device_status(tacaw_ctx *ctx, void *stream);

/* Number of kernels this context has launched since creation (bench.py's gpu_launches). */
int64_t tacaw_launch_count(const tacaw_ctx *ctx);

/* O1-O3 (PAPER.md:162 one atomic layer per slice; :219 planes at 1/4, 3/4; :505 "transmission
 * functions ... evaluated for each multislice run").
 *   n_j = clamp(floor((z_j - z0)/dz), 0, S-1)                                   (atoms outside are
 *         clamped to the first/last slice and counted -- never wrapped, :219)
 *   V_n[h,k] = sum_{j in n} f_s(q^2) exp(-2 pi i (h x_j/lx + k y_j/ly))   on in-band (h,k)
 *   v_n = Re{ IFFT2(V_n) nx ny/(lx ly) },   t_n = exp(i sigma v_n)
 * The call is batched over MD frames (same atoms, one position set per frame):
 * d_pos_A   DEVICE double [nframes][natoms][3] (Angstrom)
 * d_species DEVICE int32 [natoms] in [0,nspecies), nspecies <= 8
 * d_trans   DEVICE complex64 [nframes][nslices][ny][nx], written
 * n_clamped HOST, optional (total over the frames); when non-NULL the call synchronises the stream
 *           before returning and also returns TACAW_E_ARG if a species id was out of range (with NULL
 *           that error is sticky on the device and reported by tacaw_device_status). */
int tacaw_build_slices(tacaw_ctx *ctx, const double *d_pos_A, const int32_t *d_species, int natoms, int nframes,
                       const tacaw_species *species, double slice_thickness_A, int nslices, double z0_A,
                       void *d_trans, int *n_clamped, void *stream);

/* O4 probes: Psi0[h,k] = A exp(-2 pi i (h x_p/lx + k y_p/ly)), A = 1 iff
 * lambda^2 q^2 <= alpha^2 (alpha = 0: plane wave), inverse transformed and scaled to unit norm.
 * probe_xy_A HOST double [nprobes][2];  d_waves DEVICE complex64 [nprobes][ny][nx], written. */
int tacaw_make_probes(tacaw_ctx *ctx, const double *probe_xy_A, int nprobes, double alpha_rad,
                      void *d_waves, void *stream);

/* O5-O7 multislice ("FFTs (the core of the multislice computations)", :92, :122;
 * z-segments :72-84, :231).  For every wave w, with f = wave_frame[w]:
 *   psi <- IFFT2{ P M FFT2{ t_n psi } }  for all slices of segment 0, then segment 1, ...
 *   P[h,k] = exp(-i pi lambda dz q^2),  M = band-limit mask of the context.
 * d_waves     DEVICE complex64 [nwaves][ny][nx], overwritten with the exit waves.
 * d_probes    DEVICE complex64 [nprobes][ny][nx] or NULL.  NULL: d_waves holds the entrance waves.
 *             Non-NULL: wave w starts from d_probes[wave_probe[w]] (d_waves is output only).
 * wave_probe  HOST int32 [nwaves], values in [0, nprobes) (ignored when d_probes is NULL)
 * wave_frame  HOST int32 [nwaves], values in [0, nframes_in_flight); waves that share a frame
 *             should be adjacent (they then share each t_n read).
 * d_trans     HOST array [nframes_in_flight*nsegments] of DEVICE pointers;
 *             d_trans[f*nsegments+k] -> complex64 [nslices_per_segment[k]][ny][nx]
 * output_space 0: r-space psi_S;  1: q-space Psi_S = FFT2(psi_S), unnormalised, native FFT order. */
/* Tuning knobs of tacaw_propagate, read from the environment (defaults swept on B200):
 *   TACAW_STREAMS=n        wave groups in flight, caller's stream + n-1 internal ones (default 3; 2 from 1024^2 up; max 4;
 *                          read once)
 *   TACAW_L2_GROUP_MB=x    bytes of full waves per group (default L2/4.2 in whole row tuples, at least 3 waves; 5 waves at
 *                          1024^2, 2 waves at 2048^2)
 *   TACAW_GRID_FRAC=f      fraction of the machine-filling grid a slice-step launch uses (default 1; 0.5-1 measured equal)
 *   TACAW_PDL=0            launch the slice-step kernels without programmatic dependent launch
 * They change scheduling only, never results (tests/test_gpu_parity.py::test_propagate_l2_grouping_is_transparent). */
int tacaw_propagate(tacaw_ctx *ctx, void *d_waves, const void *d_probes, int nprobes, const int32_t *wave_probe,
                    const int32_t *wave_frame, int nwaves, const void *const *d_trans,
                    int nframes_in_flight, const int32_t *nslices_per_segment, int nsegments,
                    double slice_thickness_A, int output_space, void *stream);

/* O8 ROI map, HOST, exact: enumerate k = -ny/2..ny/2-1 (outer),
 * h = -nx/2..nx/2-1 (inner), keep by predicate, emit the native flat FFT index
 * ((k+ny)%ny)*nx + (h+nx)%nx.  idx_out NULL: count only. */
int tacaw_make_roi(const tacaw_grid *grid, double lambda_A, int mode, const double *params_rad,
                   int32_t *idx_out, int64_t *count);

/* a6 on-the-fly gather ("collects the time-consecutive exit wave functions from the
 * defined ROI", :132):  buf[p][f][r] = Psi_S(w)[roi_idx[r]] / sqrt(nx ny),  p = wave_probe[w],
 * f = wave_frame[w].
 * d_qwaves  DEVICE complex64 [nwaves][ny][nx] (q-space output of tacaw_propagate)
 * wave_probe, wave_frame  HOST int32 [nwaves] (frame = index on the time axis of d_buf)
 * d_roi_idx DEVICE int32 [nroi]
 * d_buf     DEVICE complex64 [nprobes][nframes][nroi]  (time-ordered buffer; r fastest) */
int tacaw_accumulate(tacaw_ctx *ctx, const void *d_qwaves, int nwaves, const int32_t *wave_probe,
                     const int32_t *wave_frame, const int32_t *d_roi_idx, int64_t nroi, void *d_buf,
                     int nprobes, int nframes, void *stream);

/* a5 + a6 fused ("tacaw_propagate + tacaw_accumulate may be fused internally"): the
 * same multislice run as tacaw_propagate with output_space = 1, but the LAST column kernel writes phi = Psi_S/sqrt(nx ny)
 * of the ROI pixels straight into buf[wave_probe[w]][wave_time[w]][r] -- the q-space exit wave is neither stored nor
 * re-read.  Results equal tacaw_propagate + tacaw_accumulate to fp32 rounding (one scale factor instead of two).
 * d_waves     DEVICE complex64 [nwaves][ny][nx]: scratch for the waves in flight (its content afterwards is unspecified).
 * wave_probe  HOST int32 [nwaves]: probe of each wave, in [0, nprobes_buf) (also the index into d_probes when non-NULL).
 * wave_time   HOST int32 [nwaves]: frame index of each wave on the time axis of d_buf, in [0, nframes_buf).
 * d_roi_inv   DEVICE int32 [ny][nx] from tacaw_make_roi_inverse: position r of a pixel in the ROI list, -1 outside.
 * Other arguments as tacaw_propagate / tacaw_accumulate. */
int tacaw_make_roi_inverse(tacaw_ctx *ctx, const int32_t *d_roi_idx, int64_t nroi, int32_t *d_roi_inv, void *stream);
int tacaw_propagate_accumulate(tacaw_ctx *ctx, void *d_waves, const void *d_probes, int nprobes, const int32_t *wave_probe,
                               const int32_t *wave_frame, const int32_t *wave_time, int nwaves, const void *const *d_trans,
                               int nframes_in_flight, const int32_t *nslices_per_segment, int nsegments,
                               double slice_thickness_A, const int32_t *d_roi_inv, int64_t nroi, void *d_buf,
                               int nprobes_buf, int nframes_buf, void *stream);

/* O9-O10 spectrum (Eq.(1) :37; :122, :142):
 *   Phi_k = sum_f w_f buf[p][f][r] exp(-2 pi i k f/T);  E_k = h k'/(T dt), k' = k or k-T
 *   I[p][e][r] = B(E_e/(k_B T_K)) |Phi|^2 / (T sum_f w_f^2),  B(x) = x/(1-exp(-x)), B(0) = 1
 * Energies ascending, restricted to [emin_meV, emax_meV] (inclusive, 1e-9 meV slack).
 * nframes: a power of two in [8, 2048] (register / shared-memory FFT), or any other length in [2, 512] (plain DFT over the
 * wanted energy bins -- the paper's default chunk of 200 snapshots, :164, gives its 1.4 meV sampling).
 * Series of 512 frames and more run on the single-exchange transform of the slice-step kernels; the environment variable
 * TACAW_SPEC_TWO_EXCHANGE=1 (read once) keeps the two-exchange plan of the shorter series for comparison -- same results.
 * d_I HOST-NULLABLE: pass d_I = NULL to query nE / the axis only.
 * d_I      DEVICE float [nprobes][nE][nroi];  E_axis_meV_out HOST double [>= nE] or NULL; nE HOST. */
int tacaw_spectrum(tacaw_ctx *ctx, const void *d_buf, int nprobes, int64_t nroi, int nframes, double dt_fs,
                   int window, double temperature_K, double emin_meV, double emax_meV, float *d_I,
                   double *E_axis_meV_out, int *nE, void *stream);

/* Window table, HOST, fp64 (PAPER.md:142 "multiplied by a window function before the Fourier transform", :170-182):
 * w_out[f], f = 0..n-1, for kind = TACAW_WINDOW_*; param as listed with the kinds.  Returns TACAW_E_ARG on a bad
 * kind or parameter. */
int tacaw_make_window(int kind, int n, double param, double *w_out);

/* Welch method over trajectory chunks (Eq.(2) :126):
 * the time-ordered buffer holds nframes_total stored frames.  Chunk n holds the L frames s_n + f*frame_stride,
 * f = 0..L-1 ("a stride for snapshot reading", :140), with s_0 = skip_init (Listing 1 :443
 * trajectory_chunks_skip_init: snapshots discarded as thermalisation, :164) and s_{n+1} = s_n + (L/nu)*frame_stride
 * (:138, remainder-less division, counted in the chunk's own snapshots; reading G24), for every n whose last frame
 * exists (N complete chunks):
 *   I[p][e][r] = (1/N) sum_n B(E_e/(k_B T_K)) |Phi_n|^2 / (L sum_f w_f^2),  Phi_n = DFT over the chunk of w_f buf
 * with E_k = h k'/(L dt frame_stride).  L = chunk_len: as nframes of tacaw_spectrum; nu = chunk_overlap >= 1;
 * skip_init >= 0; frame_stride >= 1.  All chunks run in ONE launch (|Phi_n|^2 summed in registers, I written once).
 * window_table HOST double [L] (tacaw_make_window or the caller's own).  N = 0 (buffer shorter than a chunk)
 * leaves d_I untouched.  nchunks HOST out (may be NULL).  Other arguments as tacaw_spectrum;
 * d_buf DEVICE complex64 [nprobes][nframes_total][nroi], d_I DEVICE float [nprobes][nE][nroi]. */
int tacaw_spectrum_welch(tacaw_ctx *ctx, const void *d_buf, int nprobes, int64_t nroi, int nframes_total, int chunk_len,
                         int chunk_overlap, int skip_init, int frame_stride, double dt_fs, const double *window_table,
                         double temperature_K, double emin_meV, double emax_meV, float *d_I, double *E_axis_meV_out, int *nE,
                         int *nchunks, void *stream);

/* DetectorSet (PAPER.md:114 "circular and annular -- with arbitrary center and radii -- and custom", :148-150, :257;
 * SURVEY.md 8(f) item 2).  Two calls:
 * tacaw_make_detector, HOST, exact: weights_out[r] = 1 if ROI pixel r lies on the detector, else 0, decided in fp64 as
 *   tx = lambda h/lx - center_rad[0], ty = lambda k/ly - center_rad[1], t2 = tx*tx + ty*ty,
 *   circular: t2 <= radii_rad[1]^2;  annular: radii_rad[0]^2 <= t2 <= radii_rad[1]^2   (both edges inclusive)
 *   with (h,k) the signed frequency indices of the native flat index roi_idx[r] (tacaw_make_roi's convention).
 * tacaw_detect, DEVICE: out[d][e][p] = sum_r weights[d][r] * I[p][e][r]  -- the energy-filtered STEM signal of
 *   detector d ("Axes of these arrays are [energy, scan-x, scan-y]", :150; p = scan position).  weights may be any
 *   caller-supplied array (the paper's "custom" detector).
 * d_I DEVICE float [nprobes][nE][nroi]; d_weights DEVICE float [ndet][nroi]; d_out DEVICE float [ndet][nE][nprobes].
 * ndet in [1, 8] per call. */
#define TACAW_DETECTOR_CIRCULAR 0
#define TACAW_DETECTOR_ANNULAR 1
int tacaw_make_detector(const tacaw_grid *grid, double lambda_A, int kind, const double *center_rad, const double *radii_rad,
                        const int32_t *roi_idx, int64_t nroi, float *weights_out);
int tacaw_detect(tacaw_ctx *ctx, const float *d_I, int nprobes, int nE, int64_t nroi, const float *d_weights, int ndet,
                 float *d_out, void *stream);

/* Scan grids ("four different scanning modes: 'unitcell', 'box', 'box_relative', and 'parallelogram'
 * ... over a two dimensional grid with grid shape defined by the user explicitly ... the end point is by design
 * not included -- 5 scan points on [0.0, 1.0) give {0.0, 0.2, 0.4, 0.6, 0.8}"; Listing 1 :416-428; SURVEY.md 8(f)
 * item 4; reading G23 of DESIGN.md).  HOST, fp64.  Point (i, j), i < shape[0], j < shape[1], is row
 * p = i*shape[1] + j of xy_out, ready for tacaw_make_probes:
 *   BOX           r = origin + (i/n0 (a_x - o_x), j/n1 (a_y - o_y)),  a = far corner of the box [A]; b, cell unused
 *   BOX_RELATIVE  the same with origin and a as fractions of the simulation cell, cell = {lx_A, ly_A}; b unused
 *   UNITCELL      r = origin + (i/n0 a_x, j/n1 a_y),  a = edge lengths of one unit cell [A]; b, cell unused
 *   PARALLELOGRAM r = origin + (i/n0) a + (j/n1) b,   a, b = edge vectors [A]; cell unused
 * xy_out HOST double [shape[0]*shape[1]][2].  Returns TACAW_E_ARG on a bad mode, a non-positive shape or a missing
 * array. */
#define TACAW_SCAN_BOX 0
#define TACAW_SCAN_BOX_RELATIVE 1
#define TACAW_SCAN_UNITCELL 2
#define TACAW_SCAN_PARALLELOGRAM 3
int tacaw_make_scan(int mode, const int32_t *shape, const double *origin, const double *a, const double *b,
                    const double *cell, double *xy_out);

/* Scan sub-batches ("scan sub-batch", Listing 1 :428 scanning_batch_shape): the scan grid is cut into tiles
 * of batch_shape[0] x batch_shape[1] points (ragged at the far edges), numbered row-major over the tile grid; tile
 * `batch` lists its scan rows p = i*shape[1] + j in ascending (i, j).  HOST.  idx_out NULL: count only.
 * nbatches (may be NULL) receives the number of tiles.  batch outside [0, nbatches) is TACAW_E_ARG. */
int tacaw_scan_batch(const int32_t *shape, const int32_t *batch_shape, int batch, int32_t *idx_out, int32_t *count,
                     int32_t *nbatches);

/* Convenience for host-resident data (bench.py's end-to-end leg): same as the calls above but the
 * named buffers are HOST memory; the library stages them through the staging region of the caller's workspace
 * (tacaw_sizes.host_staging = 1) with cudaMemcpyAsync on `stream`.  Species ids are validated on the host
 * (TACAW_E_ARG).  With n_clamped == NULL the call does not synchronise: the host arrays must then stay valid until
 * the stream has consumed them (pinned memory; pageable memory is staged by the CUDA runtime before it returns). */
int tacaw_build_slices_host(tacaw_ctx *ctx, const double *h_pos_A, const int32_t *h_species, int natoms, int nframes,
                            const tacaw_species *species, double slice_thickness_A, int nslices, double z0_A,
                            void *d_trans, int *n_clamped, void *stream);

/* tacaw_build_slices without a workspace, for callers that cannot allocate device memory (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc).  Same operation, arguments, layouts and result as
 * tacaw_build_slices (Eq.(1)-(2); O1-O3) minus n_clamped; the scratch of the binning step and
 * of K1 (clamp counter, keys, fixed-point coordinates, sorted coordinates, per-(frame, slice, species) counts and
 * offsets) lives in ONE static device array of TACAW_STATIC_SCRATCH_BYTES inside the library instead of the caller's
 * workspace, so the call works on a context that never had tacaw_set_workspace called.  Every GPU that loads the library
 * holds those 4 MiB until the process exits.  The call issues no cudaMalloc / cudaFree / allocating library routine and
 * does not synchronise; it is asynchronous on `stream`.
 * Limit: 256 + 4*(5*natoms*nframes + 2*nframes*nslices*nspecies + 2) <= TACAW_STATIC_SCRATCH_BYTES (about 200 000
 *   atom-frames); anything larger returns TACAW_E_UNSUPPORTED before any work is queued (tacaw_last_error states the
 *   bytes needed and the limit) -- use tacaw_build_slices with a workspace then.
 * Sharing: every call on a device, from any context, uses the same array, and the array keeps the last call's
 *   contents.  The counters that must start at zero are cleared on `stream` at the start of each call, so calls
 *   ordered on one stream (or ordered by events) are independent; two calls that OVERLAP on the GPU (different streams
 *   without ordering, different contexts or threads on the same device) race on the array and give undefined
 *   transmissions.  tacaw_build_slices (workspace) and this call do not share scratch.
 * Out-of-range species ids raise the context's sticky flag exactly as in tacaw_build_slices (tacaw_device_status).
 * d_pos_A, d_species, d_trans: DEVICE, caller-owned, as in tacaw_build_slices. */
#define TACAW_STATIC_SCRATCH_BYTES (4u << 20)
int tacaw_build_slices_static(tacaw_ctx *ctx, const double *d_pos_A, const int32_t *d_species, int natoms, int nframes,
                              const tacaw_species *species, double slice_thickness_A, int nslices, double z0_A,
                              void *d_trans, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* TACAW_H */

/* TACAW hot path -- fp64 CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no source, header, table or helper with the CUDA
 * library under paper_2607_02236_b200/csrc/ and neither includes the other.
 *
 * What it computes (arxiv/paper_2607_02236, "torched-TACAW"; line numbers are PAPER.md):
 *   I(q,E) ~ beta E/(1-exp(-beta E)) |phi_MD(q,E)|^2                          Eq.(1), :35-40
 *   phi_MD(q,t) = exit wave of a multislice run through MD snapshot t          :46, :92-94, :122
 *   phi_MD(q,E) = windowed time->energy Fourier transform of phi_MD(q,t)       :122, :142
 * The paper delegates the multislice formulas to the pyms library and prints none (:94); the
 * textbook scheme is used, spelled out step by step below (readings G1-G21 in DESIGN.md):
 *   O1 slice index      n_j = clamp(floor((z_j-z0)/dz), 0, S-1)
 *   O2 potential        V_n[h,k] = sum_{j in n} f_s(q^2) exp(-2 pi i (h x_j/Lx + k y_j/Ly)),
 *                       f_s(q^2) = sum_{i<4} a_si exp(-b_si q^2),  q = (h/Lx, k/Ly)
 *   O3 transmission     v_n = Re{ IFFT2(V_n) * Nx Ny/(Lx Ly) },  t_n = exp(i sigma v_n)
 *   O4 probe            Psi0[h,k] = A exp(-2 pi i (h x_p/Lx + k y_p/Ly)), A=1 iff lambda^2 q^2<=alpha^2
 *   O5 propagator       P[h,k] = exp(-i pi lambda dz q^2);  M = 1 iff q^2 <= (2/3 q_Nyq,min)^2
 *   O6 slice step       psi <- IFFT2{ P M FFT2{ t_n psi } }, n = 0..S-1, segments concatenated
 *   O7 exit wave        r-space psi_S, or q-space Psi_S = FFT2(psi_S) (unnormalised)
 *   O8 ROI map          ascending (k,h) enumeration -> native flat FFT index, int32
 *   O9 spectrum         Phi_k = sum_f w_f phi(q,t_f) exp(-2 pi i k f/T),  phi = Psi_S/sqrt(NxNy)
 *                       I = B(E_k/kBT) |Phi_k|^2 /(T sum w^2),  B(x) = x/(1-exp(-x)), B(0)=1
 *   O10 window          Hann periodic w_f = 1/2 - 1/2 cos(2 pi f/T); rect w_f = 1
 * Fourier transforms: own naive DFT for n <= 64 (or non powers of two) and own iterative
 * radix-2 FFT otherwise; no FFT/BLAS library.  Arrays are row-major [iy][ix], x fastest;
 * complex numbers are interleaved (re, im) doubles.  Forward transform has exp(-i...), the
 * inverse carries 1/(Nx Ny).
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): free-space Fresnel closed forms (P1),
 * unitarity / exact band-limit loss (P2), weak-phase closed form (P3), Bose identities (P4),
 * harmonic-mode peak bins and detailed balance (P5), single-Gaussian potential image sum (P6),
 * grid-aligned translation covariance (P7), FFT vs naive DFT vs numpy (P8), static trajectory
 * (P9), Parseval (P10), the paper's worked ROI / energy numbers (P11), segment chaining (P12),
 * O(N^4) brute force (P13).  Parity unpinned (mutual agreement only): physical sign of E (G2),
 * absolute intensity scale (G10), units of a_i (G5), the 2/3 band-limit radius (G3).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_PI 3.14159265358979323846264338327950288

static int g_fft_mode = 0; /* 0 auto (naive n<=64, radix-2 above), 1 force naive, 2 force radix-2 */

void oracle_set_fft_mode(int mode) { g_fft_mode = mode; }

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

static int signed_index(int i, int n) { return (i < n / 2) ? i : i - n; }

/* out[k] = sum_j in[j] exp(sign * 2 pi i j k / n); no scaling.  Definition of the DFT. */
void oracle_dft_naive(int n, const double *in, double *out, int sign) {
    for (int k = 0; k < n; ++k) {
        double sr = 0.0, si = 0.0;
        for (int j = 0; j < n; ++j) {
            long long m = ((long long)j * k) % n;
            double ang = sign * 2.0 * ORACLE_PI * (double)m / (double)n;
            double c = cos(ang), s = sin(ang);
            sr += in[2 * j] * c - in[2 * j + 1] * s;
            si += in[2 * j] * s + in[2 * j + 1] * c;
        }
        out[2 * k] = sr;
        out[2 * k + 1] = si;
    }
}

static int is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

/* In-place iterative radix-2 decimation-in-time FFT (bit reversal, then log2 n butterfly
 * stages); x[k] = sum_j x[j] exp(sign 2 pi i jk/n); no scaling. */
void oracle_fft_radix2(int n, double *x, int sign) {
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) {
            double tr = x[2 * i], ti = x[2 * i + 1];
            x[2 * i] = x[2 * j]; x[2 * i + 1] = x[2 * j + 1];
            x[2 * j] = tr; x[2 * j + 1] = ti;
        }
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1;
        for (int m = 0; m < half; ++m) {
            double ang = sign * 2.0 * ORACLE_PI * (double)m / (double)len;
            double wr = cos(ang), wi = sin(ang);
            for (int s = 0; s < n; s += len) {
                int p = s + m, q = p + half;
                double ur = x[2 * p], ui = x[2 * p + 1];
                double vr = x[2 * q] * wr - x[2 * q + 1] * wi;
                double vi = x[2 * q] * wi + x[2 * q + 1] * wr;
                x[2 * p] = ur + vr; x[2 * p + 1] = ui + vi;
                x[2 * q] = ur - vr; x[2 * q + 1] = ui - vi;
            }
        }
    }
}

/* 1D transform with the oracle's dispatch rule, in place, stride in complex elements. */
static void fft1d_strided(int n, double *base, long stride, int sign, double *tmp_in, double *tmp_out) {
    for (int i = 0; i < n; ++i) {
        tmp_in[2 * i] = base[2 * i * stride];
        tmp_in[2 * i + 1] = base[2 * i * stride + 1];
    }
    int naive = (g_fft_mode == 1) || (g_fft_mode == 0 && n <= 64) || !is_pow2(n);
    const double *res;
    if (naive) {
        oracle_dft_naive(n, tmp_in, tmp_out, sign);
        res = tmp_out;
    } else {
        oracle_fft_radix2(n, tmp_in, sign);
        res = tmp_in;
    }
    for (int i = 0; i < n; ++i) {
        base[2 * i * stride] = res[2 * i];
        base[2 * i * stride + 1] = res[2 * i + 1];
    }
}

void oracle_fft1d(int n, double *x, int sign) {
    double *ti = (double *)malloc(sizeof(double) * 4 * (size_t)n);
    fft1d_strided(n, x, 1, sign, ti, ti + 2 * n);
    free(ti);
}

/* 2D transform of a[ny][nx] in place: all rows (x), then all columns (y).
 * sign=-1 forward (no scaling); sign=+1 inverse (scaled by 1/(nx ny)). */
void oracle_fft2(int ny, int nx, double *a, int sign) {
    int nmax = nx > ny ? nx : ny;
    /* rows, then columns: independent 1D transforms, shared out over threads when the caller is not already
     * running in parallel (the arithmetic of each transform is untouched) */
    int par = 1;
#ifdef _OPENMP
    par = !omp_in_parallel() && (size_t)nx * ny >= 65536;
#endif
#pragma omp parallel if (par)
    {
        double *tmp = (double *)malloc(sizeof(double) * 4 * (size_t)nmax);
#pragma omp for schedule(static)
        for (int iy = 0; iy < ny; ++iy) fft1d_strided(nx, a + 2 * (size_t)iy * nx, 1, sign, tmp, tmp + 2 * nmax);
#pragma omp for schedule(static)
        for (int ix = 0; ix < nx; ++ix) fft1d_strided(ny, a + 2 * (size_t)ix, nx, sign, tmp, tmp + 2 * nmax);
        free(tmp);
    }
    if (sign > 0) {
        double s = 1.0 / ((double)nx * (double)ny);
        for (size_t i = 0; i < 2 * (size_t)nx * ny; ++i) a[i] *= s;
    }
}

/* O5 mask: M[h,k] = 1 iff q^2 <= (2/3)^2 min(Nx/(2Lx), Ny/(2Ly))^2.  For a square cell this is
 * the integer test 9(h^2+k^2) <= N^2. */
static int in_band(int h, int k, int nx, int ny, double lx, double ly, int bandlimit) {
    if (!bandlimit) return 1;
    if (nx == ny && lx == ly) return 9LL * ((long long)h * h + (long long)k * k) <= (long long)nx * nx;
    double qx = h / lx, qy = k / ly;
    double qn = fmin(nx / (2.0 * lx), ny / (2.0 * ly));
    return qx * qx + qy * qy <= (4.0 / 9.0) * qn * qn;
}

/* O1-O3.  pos [natoms][3] (A), species [natoms], a/b [nspecies][4].
 * bandlimit=1: V only where M=1 (reading G4); bandlimit=0 ("pot_full"): all |h|<nx/2, |k|<ny/2.
 * pot_mode=0: every term exp(-2 pi i(h x/Lx + k y/Ly)) evaluated directly (the definition);
 * pot_mode=1: the same term as the product exp(-2 pi i h x/Lx) * exp(-2 pi i k y/Ly) of two
 *             per-atom phase tables (an exact identity; pinned against mode 0 in the tests).
 * Outputs (any may be NULL): trans [S][ny][nx] complex, v [S][ny][nx] real, Vq [S][ny][nx] complex,
 * n_clamped, max_imag (max |Im v| / max |Re v| over all slices). */
int oracle_build_slices(int nx, int ny, double lx, double ly, const double *pos, const int32_t *species,
                        int natoms, int nspecies, const double *a, const double *b, double dz, int nslices,
                        double z0, double sigma, int bandlimit, int pot_mode, double *trans, double *v_out,
                        double *vq_out, int *n_clamped, double *max_imag) {
    if (nx <= 0 || ny <= 0 || nslices <= 0 || natoms < 0) return -1;
    int *slice_of = (int *)malloc(sizeof(int) * (size_t)(natoms > 0 ? natoms : 1));
    int clamped = 0;
    for (int j = 0; j < natoms; ++j) {
        if (species[j] < 0 || species[j] >= nspecies) { free(slice_of); return -2; }
        double f = floor((pos[3 * j + 2] - z0) / dz);
        int n;
        if (f < 0.0) { n = 0; ++clamped; }
        else if (f > (double)(nslices - 1)) { n = nslices - 1; ++clamped; }
        else n = (int)f;
        slice_of[j] = n;
    }
    if (n_clamped) *n_clamped = clamped;
    size_t npix = (size_t)nx * ny;
    /* f_s(q^2) depends on the species and the pixel only, not on the atom: evaluated once per (species, pixel) with the
     * same expression and used for every atom of that species below (a table of the values, no change of arithmetic) */
    double *ftab = (double *)calloc((size_t)(nspecies > 0 ? nspecies : 1) * npix, sizeof(double));
    unsigned char *carries = (unsigned char *)calloc(npix, 1);   /* 1 where V is defined: in band, not on a Nyquist line */
#pragma omp parallel for schedule(static)
    for (int iy = 0; iy < ny; ++iy) {
        int k = signed_index(iy, ny);
        for (int ix = 0; ix < nx; ++ix) {
            int h = signed_index(ix, nx);
            carries[(size_t)iy * nx + ix] = (2 * k != -ny) && (2 * h != -nx) && in_band(h, k, nx, ny, lx, ly, bandlimit);
            double q2 = (h / lx) * (h / lx) + (k / ly) * (k / ly);
            for (int sidx = 0; sidx < nspecies; ++sidx) {
                const double *as = a + 4 * sidx, *bs = b + 4 * sidx;
                double f = 0.0;
                for (int i = 0; i < 4; ++i) f += as[i] * exp(-bs[i] * q2);
                ftab[(size_t)sidx * npix + (size_t)iy * nx + ix] = f;
            }
        }
    }
    double worst_ratio = 0.0;
    /* slices are independent: one thread per slice when there are enough of them; otherwise the slices run one after the
     * other and the rows of each atom's contribution are shared out instead (every pixel still adds its atoms in the same
     * order, so the sums are unchanged) */
    int over_slices = 1;
#ifdef _OPENMP
    over_slices = nslices >= omp_get_max_threads();
#endif
#pragma omp parallel for schedule(dynamic, 1) reduction(max : worst_ratio) if (over_slices)
    for (int n = 0; n < nslices; ++n) {
        double *V = (double *)calloc(2 * npix, sizeof(double));
        double *ex = (double *)malloc(sizeof(double) * 2 * (size_t)nx);
        double *ey = (double *)malloc(sizeof(double) * 2 * (size_t)ny);
        for (int j = 0; j < natoms; ++j) {
            if (slice_of[j] != n) continue;
            const double *fs = ftab + (size_t)species[j] * npix;
            double xf = pos[3 * j] / lx, yf = pos[3 * j + 1] / ly;
            if (pot_mode == 1) {
                for (int ix = 0; ix < nx; ++ix) {
                    double ang = -2.0 * ORACLE_PI * signed_index(ix, nx) * xf;
                    ex[2 * ix] = cos(ang); ex[2 * ix + 1] = sin(ang);
                }
                for (int iy = 0; iy < ny; ++iy) {
                    double ang = -2.0 * ORACLE_PI * signed_index(iy, ny) * yf;
                    ey[2 * iy] = cos(ang); ey[2 * iy + 1] = sin(ang);
                }
            }
#pragma omp parallel for schedule(static) if (!over_slices)
            for (int iy = 0; iy < ny; ++iy) {
                int k = signed_index(iy, ny);
                for (int ix = 0; ix < nx; ++ix) {
                    int h = signed_index(ix, nx);
                    if (!carries[(size_t)iy * nx + ix]) continue;   /* Nyquist lines and out-of-band pixels carry no V */
                    double f = fs[(size_t)iy * nx + ix];
                    double pr, pi_;
                    if (pot_mode == 1) {
                        pr = ex[2 * ix] * ey[2 * iy] - ex[2 * ix + 1] * ey[2 * iy + 1];
                        pi_ = ex[2 * ix] * ey[2 * iy + 1] + ex[2 * ix + 1] * ey[2 * iy];
                    } else {
                        double ang = -2.0 * ORACLE_PI * (h * xf + k * yf);
                        pr = cos(ang); pi_ = sin(ang);
                    }
                    V[2 * ((size_t)iy * nx + ix)] += f * pr;
                    V[2 * ((size_t)iy * nx + ix) + 1] += f * pi_;
                }
            }
        }
        if (vq_out) memcpy(vq_out + 2 * npix * n, V, sizeof(double) * 2 * npix);
        oracle_fft2(ny, nx, V, +1);
        double scale = ((double)nx * (double)ny) / (lx * ly);
        double mre = 0.0, mim = 0.0;
        for (size_t i = 0; i < npix; ++i) {
            double vr = V[2 * i] * scale, vi = V[2 * i + 1] * scale;
            if (fabs(vr) > mre) mre = fabs(vr);
            if (fabs(vi) > mim) mim = fabs(vi);
            if (v_out) v_out[npix * n + i] = vr;
            if (trans) {
                trans[2 * (npix * n + i)] = cos(sigma * vr);
                trans[2 * (npix * n + i) + 1] = sin(sigma * vr);
            }
        }
        double ratio = (mre > 0.0) ? mim / mre : 0.0;
        if (ratio > worst_ratio) worst_ratio = ratio;
        free(V); free(ex); free(ey);
    }
    if (max_imag) *max_imag = worst_ratio;
    free(slice_of);
    free(ftab);
    free(carries);
    return 0;
}

/* O4.  probe_xy [nprobes][2] (A); alpha in rad (0 -> plane wave: only (0,0) passes);
 * waves [nprobes][ny][nx] complex, unit norm. */
int oracle_make_probes(int nx, int ny, double lx, double ly, double lambda, const double *probe_xy,
                       int nprobes, double alpha, double *waves) {
    size_t npix = (size_t)nx * ny;
#pragma omp parallel for schedule(dynamic, 1)
    for (int p = 0; p < nprobes; ++p) {
        double *w = waves + 2 * npix * p;
        double xp = probe_xy[2 * p], yp = probe_xy[2 * p + 1];
        for (int iy = 0; iy < ny; ++iy) {
            int k = signed_index(iy, ny);
            for (int ix = 0; ix < nx; ++ix) {
                int h = signed_index(ix, nx);
                double q2 = (h / lx) * (h / lx) + (k / ly) * (k / ly);
                size_t i = (size_t)iy * nx + ix;
                if (lambda * lambda * q2 <= alpha * alpha) {
                    double ang = -2.0 * ORACLE_PI * (h * xp / lx + k * yp / ly);
                    w[2 * i] = cos(ang); w[2 * i + 1] = sin(ang);
                } else {
                    w[2 * i] = 0.0; w[2 * i + 1] = 0.0;
                }
            }
        }
        oracle_fft2(ny, nx, w, +1);
        double s = 0.0;
        for (size_t i = 0; i < 2 * npix; ++i) s += w[i] * w[i];
        double inv = 1.0 / sqrt(s);
        for (size_t i = 0; i < 2 * npix; ++i) w[i] *= inv;
    }
    return 0;
}

/* O5-O7.  waves [nwaves][ny][nx] complex, in place.  wave_frame[w] = in-flight frame index f.
 * trans[f*nsegments + k] -> complex [nslices_per_segment[k]][ny][nx].
 * output_space 0: r-space psi_S; 1: q-space FFT2(psi_S), unnormalised, native FFT order.
 * norms (optional) [nwaves][total_slices+1]: sum |psi|^2 before the first and after every step. */
int oracle_propagate(int nx, int ny, double lx, double ly, double lambda, int bandlimit, double *waves,
                     const int32_t *wave_frame, int nwaves, const double *const *trans, int nframes,
                     const int32_t *nslices_per_segment, int nsegments, double dz, int output_space,
                     double *norms) {
    size_t npix = (size_t)nx * ny;
    int total = 0;
    for (int k = 0; k < nsegments; ++k) total += nslices_per_segment[k];
    double *P = (double *)malloc(sizeof(double) * 2 * npix);
    for (int iy = 0; iy < ny; ++iy) {
        int k = signed_index(iy, ny);
        for (int ix = 0; ix < nx; ++ix) {
            int h = signed_index(ix, nx);
            size_t i = (size_t)iy * nx + ix;
            double q2 = (h / lx) * (h / lx) + (k / ly) * (k / ly);
            if (in_band(h, k, nx, ny, lx, ly, bandlimit)) {
                double ang = -ORACLE_PI * lambda * dz * q2;
                P[2 * i] = cos(ang); P[2 * i + 1] = sin(ang);
            } else {
                P[2 * i] = 0.0; P[2 * i + 1] = 0.0;
            }
        }
    }
    int bad = 0;
    /* waves are independent: one thread per wave when there are enough of them, otherwise the waves run one after
     * the other and each 2D transform is shared out over the threads instead (oracle_fft2) */
    int over_waves = 1;
#ifdef _OPENMP
    over_waves = nwaves >= omp_get_max_threads();
#endif
#pragma omp parallel for schedule(dynamic, 1) if (over_waves)
    for (int w = 0; w < nwaves; ++w) {
        double *psi = waves + 2 * npix * w;
        int f = wave_frame ? wave_frame[w] : 0;
        if (f < 0 || f >= nframes) { bad = 1; continue; }
        int step = 0;
        if (norms) {
            double s = 0.0;
            for (size_t i = 0; i < 2 * npix; ++i) s += psi[i] * psi[i];
            norms[(size_t)w * (total + 1)] = s;
        }
        for (int k = 0; k < nsegments; ++k) {
            const double *tseg = trans[(size_t)f * nsegments + k];
            for (int n = 0; n < nslices_per_segment[k]; ++n, ++step) {
                const double *t = tseg + 2 * npix * n;
                for (size_t i = 0; i < npix; ++i) {
                    double pr = psi[2 * i], pi_ = psi[2 * i + 1];
                    psi[2 * i] = pr * t[2 * i] - pi_ * t[2 * i + 1];
                    psi[2 * i + 1] = pr * t[2 * i + 1] + pi_ * t[2 * i];
                }
                oracle_fft2(ny, nx, psi, -1);
                for (size_t i = 0; i < npix; ++i) {
                    double pr = psi[2 * i], pi_ = psi[2 * i + 1];
                    psi[2 * i] = pr * P[2 * i] - pi_ * P[2 * i + 1];
                    psi[2 * i + 1] = pr * P[2 * i + 1] + pi_ * P[2 * i];
                }
                oracle_fft2(ny, nx, psi, +1);
                if (norms) {
                    double s = 0.0;
                    for (size_t i = 0; i < 2 * npix; ++i) s += psi[i] * psi[i];
                    norms[(size_t)w * (total + 1) + step + 1] = s;
                }
            }
        }
        if (output_space == 1) oracle_fft2(ny, nx, psi, -1);
    }
    free(P);
    return bad ? -3 : 0;
}

/* O8.  mode 0 full, 1 disc (params: theta_o), 2 annulus (theta_i, theta_o), 3 rect
 * (xmin, xmax, ymin, ymax) -- all in rad.  idx_out NULL -> count only. */
int oracle_make_roi(int nx, int ny, double lx, double ly, double lambda, int mode, const double *params,
                    int32_t *idx_out, int64_t *count) {
    int64_t c = 0;
    int square = (nx == ny && lx == ly);
    for (int k = -ny / 2; k < ny - ny / 2; ++k) {
        for (int h = -nx / 2; h < nx - nx / 2; ++h) {
            int keep;
            if (mode == 0) keep = 1;
            else if (mode == 1 || mode == 2) {
                double t2;
                if (square) {
                    double s = lambda / lx;
                    t2 = s * s * (double)((long long)h * h + (long long)k * k);
                } else {
                    t2 = lambda * lambda * ((h / lx) * (h / lx) + (k / ly) * (k / ly));
                }
                double to = (mode == 1) ? params[0] : params[1];
                keep = t2 <= to * to;
                if (mode == 2) keep = keep && (t2 >= params[0] * params[0]);
            } else if (mode == 3) {
                double tx = lambda * h / lx, ty = lambda * k / ly;
                keep = tx >= params[0] && tx <= params[1] && ty >= params[2] && ty <= params[3];
            } else return -1;
            if (keep) {
                if (idx_out) idx_out[c] = (int32_t)(((k + ny) % ny) * nx + (h + nx) % nx);
                ++c;
            }
        }
    }
    *count = c;
    return 0;
}

/* a6.  qwaves [nwaves][ny][nx] complex (q-space, unnormalised).  buf [nprobes][nframes][nroi]
 * complex: buf[p][f][r] = qwaves[w][idx[r]] / sqrt(nx ny) with p = wave_probe[w], f = wave_frame[w]. */
int oracle_accumulate(int nx, int ny, const double *qwaves, int nwaves, const int32_t *wave_probe,
                      const int32_t *wave_frame, const int32_t *roi_idx, int64_t nroi, double *buf,
                      int nprobes, int nframes) {
    size_t npix = (size_t)nx * ny;
    double s = 1.0 / sqrt((double)nx * (double)ny);
    for (int w = 0; w < nwaves; ++w) {
        int p = wave_probe[w], f = wave_frame[w];
        if (p < 0 || p >= nprobes || f < 0 || f >= nframes) return -3;
        double *dst = buf + 2 * (((size_t)p * nframes + f) * (size_t)nroi);
        const double *src = qwaves + 2 * npix * w;
        for (int64_t r = 0; r < nroi; ++r) {
            dst[2 * r] = src[2 * (size_t)roi_idx[r]] * s;
            dst[2 * r + 1] = src[2 * (size_t)roi_idx[r] + 1] * s;
        }
    }
    return 0;
}

/* O9 Bose / detailed-balance factor B(x) = x/(1-exp(-x)), B(0) = 1. */
double oracle_bose(double x) {
    if (x == 0.0) return 1.0;
    return x / (-expm1(-x));
}

/* O10. window 0 rect, 1 Hann (periodic). */
void oracle_window(int window, int nframes, double *w) {
    for (int f = 0; f < nframes; ++f)
        w[f] = (window == 1) ? 0.5 - 0.5 * cos(2.0 * ORACLE_PI * (double)f / (double)nframes) : 1.0;
}

/* Energy axis (ascending) inside [emin, emax] (inclusive, 1e-9 meV slack): returns count, fills
 * E (meV) and the DFT bin k in [0,T) of each kept energy. */
int oracle_energy_axis(int nframes, double dt_fs, double emin, double emax, double *E, int32_t *bins) {
    const double h_mev_fs = 4135.667696;
    int c = 0;
    for (int kp = -nframes / 2; kp < nframes - nframes / 2; ++kp) {
        double e = h_mev_fs * (double)kp / ((double)nframes * dt_fs);
        if (e < emin - 1e-9 || e > emax + 1e-9) continue;
        if (E) E[c] = e;
        if (bins) bins[c] = (kp + nframes) % nframes;
        ++c;
    }
    return c;
}

/* O9 with the window given as a table w[nframes], on frames
 * [frame0, frame0 + nframes) of a buffer [nprobes][nframes_total][nroi]; I [nprobes][nE][nroi] (double), E_out [nE]. */
int oracle_spectrum_table(const double *buf, int nprobes, int64_t nroi, int nframes_total, int frame0, int nframes, double dt_fs,
                          const double *w, double temperature_K, double emin, double emax, double *I, double *E_out,
                          int *nE_out) {
    const double kb_mev = 8.617333262e-5 * 1e3;
    int nE = oracle_energy_axis(nframes, dt_fs, emin, emax, NULL, NULL);
    if (nE_out) *nE_out = nE;
    if (!I) return 0;
    double *E = (double *)malloc(sizeof(double) * (size_t)(nE > 0 ? nE : 1));
    int32_t *bins = (int32_t *)malloc(sizeof(int32_t) * (size_t)(nE > 0 ? nE : 1));
    oracle_energy_axis(nframes, dt_fs, emin, emax, E, bins);
    if (E_out) memcpy(E_out, E, sizeof(double) * (size_t)nE);
    double sw2 = 0.0;
    for (int f = 0; f < nframes; ++f) sw2 += w[f] * w[f];
    double norm = 1.0 / ((double)nframes * sw2);
    int64_t nser = (int64_t)nprobes * nroi;
#pragma omp parallel
    {
        double *x = (double *)malloc(sizeof(double) * 6 * (size_t)nframes);
#pragma omp for schedule(static)
        for (int64_t s = 0; s < nser; ++s) {
            int64_t p = s / nroi, r = s % nroi;
            for (int f = 0; f < nframes; ++f) {
                const double *src = buf + 2 * ((p * nframes_total + frame0 + f) * nroi + r);
                x[2 * f] = w[f] * src[0];
                x[2 * f + 1] = w[f] * src[1];
            }
            fft1d_strided(nframes, x, 1, -1, x + 2 * nframes, x + 4 * nframes);
            for (int e = 0; e < nE; ++e) {
                double re = x[2 * bins[e]], im = x[2 * bins[e] + 1];
                I[(p * nE + e) * nroi + r] = oracle_bose(E[e] / (kb_mev * temperature_K)) * (re * re + im * im) * norm;
            }
        }
        free(x);
    }
    free(E); free(bins);
    return 0;
}

/* O9.  buf [nprobes][nframes][nroi] complex -> I [nprobes][nE][nroi] (double).  E_out [nE].  window: O10. */
int oracle_spectrum(const double *buf, int nprobes, int64_t nroi, int nframes, double dt_fs, int window,
                    double temperature_K, double emin, double emax, double *I, double *E_out, int *nE_out) {
    double *w = (double *)malloc(sizeof(double) * (size_t)nframes);
    oracle_window(window, nframes, w);
    int rc = oracle_spectrum_table(buf, nprobes, nroi, nframes, 0, nframes, dt_fs, w, temperature_K, emin, emax, I, E_out, nE_out);
    free(w);
    return rc;
}

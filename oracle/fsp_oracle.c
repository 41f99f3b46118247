/*
 * fsp_oracle.c -- CPU ORACLE for the free-space Poisson convolution of
 * arxiv 2405.02603 (Mayani et al.), Hockney-Eastwood (HE) and Vico-Greengard (VG).
 *
 * THIS FILE IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, the smoke check in
 * __graft_entry__.py and bench.py's cpu_baseline / --impl reference legs may build, load or
 * call it.  It shares no code, header, table or constant generator with the CUDA path under
 * paper_2405_02603_b200/csrc/.  It is plain, slow and written to be checked against the paper
 * by eye: no pruning, no fusion, no blocking -- the paper's steps in the paper's order.
 *
 * Citations are PAPER.md:<line> (= /root/reference/PAPER.md) and DESIGN.md "Readings" R<n>.
 *
 *   orc_direct_sum*      PAPER.md:35   "discretizing G and rho on the computational mesh, and
 *                                        approximating the integral as a sum" (+ weight hxhyhz of
 *                                        PAPER.md:80).  THE plain definition (Def. O1); long double sums.
 *   orc_green_table_vg_entries  PAPER.md:100-102  single entries of the VG table by the explicit triple
 *                                        cosine sum (no transform): the reference for tables at full size.
 *   orc_fft_radix2 /     PAPER.md:37   the Fourier transform F; textbook iterative radix-2
 *   orc_dft_direct                      Cooley-Tukey and the O(n^2) definition of the DFT.
 *   orc_green_table_he   PAPER.md:35,72-76  G = 1/(4 pi |x|), regularised at the origin (R5).
 *   orc_green_table_vg   PAPER.md:88-98     Eq. 3 on the 4N grid, inverse DFT, restricted.
 *   orc_green_table_vg2  PAPER.md:100-102,205  same values on the (2N+1)^3 grid, DCT-I.
 *   orc_green_table_vgm / orc_vg_safe_factors   the same with per-axis oversampling m_d (8(f) N2, R17).
 *   orc_green_g2 /       PAPER.md:72-74  the 8-case mirror G2 on the doubled grid, and its DFT.
 *   orc_green_spectrum
 *   orc_solve            PAPER.md:67-82  steps 1-5: double, zero-pad, FFT, multiply, inverse FFT,
 *                                        scale by hxhyhz, restrict.
 *   orc_solve_field      PAPER.md:227-231 (Eq. A.1)  E = -grad phi, spectral gradient on the doubled
 *                                        grid (8(f) N3, R18): steps 1-4, times -i k_d, inverse FFT, restrict.
 *   orc_solve_mixed /    PAPER.md:67, 72  periodic directions (8(f) N4, R20): "double the computational grid in the
 *   orc_direct_sum_mixed                 non-periodic directions" only; G made periodic along a periodic direction
 *                                        with the period of the domain (nearest image); the same sum written out.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): numpy brute force on tiny grids, numpy.fft on
 * random vectors, the closed-form Gaussian potential with second-order (HE) and
 * spectral (VG) convergence, delta-source => table, VG plain == VG modified, far field -> 1/(4 pi r).
 * No function here is "parity unpinned" except the sign of the HE origin value g0 (R5), which is a
 * parameter.
 *
 * Layout: every 3-D array is C order, last index fastest.  Complex arrays are interleaved
 * (re, im) doubles, i.e. numpy complex128.  All arithmetic is fp64.
 * OpenMP (if compiled with -fopenmp) only distributes independent pencils / output points.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_OK 0
#define ORC_EINVAL -1
#define ORC_ENOMEM -2

static const double ORC_PI = 3.14159265358979323846264338327950288;

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

static int is_pow2(long n) { return n > 0 && (n & (n - 1)) == 0; }

/* ------------------------------------------------------------------------------------------
 * 1-D transforms.  sign = -1: X[k] = sum_n x[n] exp(-2 pi i k n / n_len)   (forward, F)
 *                  sign = +1: X[k] = sum_n x[n] exp(+2 pi i k n / n_len)   (inverse, NOT scaled)
 * The 1/n of F^-1 is applied by the callers, so that F^-1 F = I (R7).
 * ------------------------------------------------------------------------------------------ */

/* The definition of the DFT, O(n^2).  in/out: n complex (interleaved), must not alias. */
void orc_dft_direct(long n, const double* in, double* out, int sign) {
    for (long k = 0; k < n; ++k) {
        double sr = 0.0, si = 0.0;
        for (long m = 0; m < n; ++m) {
            /* reduce k*m mod n before the trig call so the argument stays in [0, 2 pi) */
            long km = (long)(((int64_t)k * (int64_t)m) % (int64_t)n);
            double ang = (double)sign * 2.0 * ORC_PI * (double)km / (double)n;
            double c = cos(ang), s = sin(ang);
            double xr = in[2 * m], xi = in[2 * m + 1];
            sr += xr * c - xi * s;
            si += xr * s + xi * c;
        }
        out[2 * k] = sr;
        out[2 * k + 1] = si;
    }
}

/* Textbook iterative radix-2 decimation-in-time Cooley-Tukey FFT, in place, n a power of two:
 * bit-reversal permutation, then log2(n) butterfly passes.  Each twiddle is taken from cos/sin
 * directly (no recurrence), so the error stays O(eps log n). */
void orc_fft_radix2(long n, double* a, int sign) {
    /* bit reversal */
    for (long i = 1, j = 0; i < n; ++i) {
        long bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) {
            double tr = a[2 * i], ti = a[2 * i + 1];
            a[2 * i] = a[2 * j];
            a[2 * i + 1] = a[2 * j + 1];
            a[2 * j] = tr;
            a[2 * j + 1] = ti;
        }
    }
    for (long len = 2; len <= n; len <<= 1) {
        long half = len >> 1;
        for (long j = 0; j < half; ++j) {
            double ang = (double)sign * 2.0 * ORC_PI * (double)j / (double)len;
            double wr = cos(ang), wi = sin(ang);
            for (long i = j; i < n; i += len) {
                long p = i + half;
                double ur = a[2 * i], ui = a[2 * i + 1];
                double vr = a[2 * p] * wr - a[2 * p + 1] * wi;
                double vi = a[2 * p] * wi + a[2 * p + 1] * wr;
                a[2 * i] = ur + vr;
                a[2 * i + 1] = ui + vi;
                a[2 * p] = ur - vr;
                a[2 * p + 1] = ui - vi;
            }
        }
    }
}

/* One 1-D transform of length n, in place.  method 0: radix-2 if n is a power of two, else the
 * direct definition; method 1: always the direct definition. */
static void fft1d(long n, double* a, double* tmp, int sign, int method) {
    if (method == 0 && is_pow2(n)) {
        orc_fft_radix2(n, a, sign);
    } else {
        orc_dft_direct(n, a, tmp, sign);
        memcpy(a, tmp, sizeof(double) * 2 * (size_t)n);
    }
}

/* Exposed for the pins: transform one vector (out of place). */
int orc_fft1d(long n, const double* in, double* out, int sign, int method) {
    if (n < 1 || !in || !out || (sign != 1 && sign != -1)) return ORC_EINVAL;
    double* tmp = (double*)malloc(sizeof(double) * 2 * (size_t)n);
    if (!tmp) return ORC_ENOMEM;
    memcpy(out, in, sizeof(double) * 2 * (size_t)n);
    fft1d(n, out, tmp, sign, method);
    free(tmp);
    return ORC_OK;
}

/* Separable 3-D DFT, in place, on a complex array a[n0][n1][n2]: 1-D transforms along axis 2,
 * then axis 1, then axis 0 (each pencil gathered into a contiguous buffer, transformed, scattered
 * back).  Unscaled for both signs. */
int orc_fft3d(long n0, long n1, long n2, double* a, int sign, int method) {
    if (n0 < 1 || n1 < 1 || n2 < 1 || !a || (sign != 1 && sign != -1)) return ORC_EINVAL;
    long dims[3] = {n0, n1, n2};
    long strides[3] = {n1 * n2, n2, 1};
    int err = 0;
    for (int axis = 2; axis >= 0; --axis) {
        long n = dims[axis], st = strides[axis];
        int o1 = (axis + 1) % 3, o2 = (axis + 2) % 3;
        long m1 = dims[o1], m2 = dims[o2], s1 = strides[o1], s2 = strides[o2];
#pragma omp parallel
        {
            double* buf = (double*)malloc(sizeof(double) * 4 * (size_t)n);
            if (!buf) {
#pragma omp atomic write
                err = 1;
            }
#pragma omp for collapse(2) schedule(static)
            for (long i1 = 0; i1 < m1; ++i1) {
                for (long i2 = 0; i2 < m2; ++i2) {
                    if (!buf) continue;
                    double* base = a + 2 * (i1 * s1 + i2 * s2);
                    for (long i = 0; i < n; ++i) {
                        buf[2 * i] = base[2 * i * st];
                        buf[2 * i + 1] = base[2 * i * st + 1];
                    }
                    fft1d(n, buf, buf + 2 * n, sign, method);
                    for (long i = 0; i < n; ++i) {
                        base[2 * i * st] = buf[2 * i];
                        base[2 * i * st + 1] = buf[2 * i + 1];
                    }
                }
            }
            free(buf);
        }
        if (err) return ORC_ENOMEM;
    }
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------------
 * Green's-function tables.  T[dx][dy][dz], 0 <= d_d <= N_d, is the real-space kernel at the
 * displacement (dx hx, dy hy, dz hz); shape (Nx+1, Ny+1, Nz+1).
 * ------------------------------------------------------------------------------------------ */

/* HE: G(x) = 1/(4 pi |x|), with the singular origin value replaced by g0
 * (reading R5: g0 = +1/(4 pi) by default, passed in by the caller). */
int orc_green_table_he(long Nx, long Ny, long Nz, const double h[3], double g0, double* T) {
    if (Nx < 1 || Ny < 1 || Nz < 1 || !h || !T || !(h[0] > 0) || !(h[1] > 0) || !(h[2] > 0))
        return ORC_EINVAL;
    for (long dx = 0; dx <= Nx; ++dx)
        for (long dy = 0; dy <= Ny; ++dy)
            for (long dz = 0; dz <= Nz; ++dz) {
                double x = dx * h[0], y = dy * h[1], z = dz * h[2];
                double r = sqrt(x * x + y * y + z * z);
                double g = (dx == 0 && dy == 0 && dz == 0) ? g0 : 1.0 / (4.0 * ORC_PI * r);
                T[(dx * (Ny + 1) + dy) * (Nz + 1) + dz] = g;
            }
    return ORC_OK;
}

/* Eq. 3: G_L(s) = 2 (sin(L|s|/2)/|s|)^2, with the s -> 0 limit L^2/2 (R8). */
static double vg_GL(double sx, double sy, double sz, double L) {
    double s = sqrt(sx * sx + sy * sy + sz * sz);
    if (s == 0.0) return 0.5 * L * L;
    double q = sin(0.5 * L * s) / s;
    return 2.0 * q * q;
}

/* Truncation window L = alpha sqrt(Lx^2+Ly^2+Lz^2), L_d = N_d h_d. */
double orc_vg_window(long Nx, long Ny, long Nz, const double h[3], double alpha) {
    double Lx = Nx * h[0], Ly = Ny * h[1], Lz = Nz * h[2];
    return alpha * sqrt(Lx * Lx + Ly * Ly + Lz * Lz);
}

/* VG, plain precompute (reading R9):
 *  1. M_d = 4 N_d points per axis; frequencies in DFT order k_d in {0..2N_d-1, -2N_d..-1},
 *     s_d = 2 pi k_d / (M_d h_d).
 *  2. fill G_L(s) on the (4N)^3 grid.
 *  3. inverse DFT, as the Riemann sum of (2 pi)^-3 int G_L e^{i s.x} ds with ds_d = 2 pi/(M_d h_d):
 *       G4[n] = 1/prod_d(M_d h_d) * sum_k G_L(s_k) exp(+2 pi i sum_d k_d n_d / M_d).
 *  4. restrict: T[d] = Re G4[d], 0 <= d_d <= N_d.
 * Needs a (4N)^3 complex array (the memory cost the paper talks about). */
int orc_green_table_vg(long Nx, long Ny, long Nz, const double h[3], double alpha, int method,
                       double* T) {
    if (Nx < 1 || Ny < 1 || Nz < 1 || !h || !T || !(h[0] > 0) || !(h[1] > 0) || !(h[2] > 0) ||
        !(alpha > 0))
        return ORC_EINVAL;
    long Mx = 4 * Nx, My = 4 * Ny, Mz = 4 * Nz;
    double L = orc_vg_window(Nx, Ny, Nz, h, alpha);
    size_t total = (size_t)Mx * My * Mz;
    double* g = (double*)malloc(sizeof(double) * 2 * total);
    if (!g) return ORC_ENOMEM;
#pragma omp parallel for schedule(static)
    for (long ix = 0; ix < Mx; ++ix) {
        long kx = ix < 2 * Nx ? ix : ix - Mx;
        double sx = 2.0 * ORC_PI * kx / (Mx * h[0]);
        for (long iy = 0; iy < My; ++iy) {
            long ky = iy < 2 * Ny ? iy : iy - My;
            double sy = 2.0 * ORC_PI * ky / (My * h[1]);
            for (long iz = 0; iz < Mz; ++iz) {
                long kz = iz < 2 * Nz ? iz : iz - Mz;
                double sz = 2.0 * ORC_PI * kz / (Mz * h[2]);
                size_t o = ((size_t)ix * My + iy) * Mz + iz;
                g[2 * o] = vg_GL(sx, sy, sz, L);
                g[2 * o + 1] = 0.0;
            }
        }
    }
    int rc = orc_fft3d(Mx, My, Mz, g, +1, method);
    if (rc != ORC_OK) {
        free(g);
        return rc;
    }
    double scale = 1.0 / ((Mx * h[0]) * (My * h[1]) * (Mz * h[2]));
    for (long dx = 0; dx <= Nx; ++dx)
        for (long dy = 0; dy <= Ny; ++dy)
            for (long dz = 0; dz <= Nz; ++dz) {
                size_t o = ((size_t)dx * My + dy) * Mz + dz;
                T[(dx * (Ny + 1) + dy) * (Nz + 1) + dz] = scale * g[2 * o];
            }
    free(g);
    return ORC_OK;
}

/* Un-normalised DCT-I of size n+1 along one axis (FFTW's REDFT00 convention):
 *     out[d] = sum_{k=0..n} w_k in[k] cos(pi k d / n),   w_0 = w_n = 1, w_k = 2 otherwise,
 * for d = 0..nout-1 (nout <= n+1).  This is the DFT of length 2n of the even extension of `in`
 * ("the discrete Fourier transform reduces to a discrete cosine transform" for a
 * real, even signal; type 1).
 *   method 1: the cosine sum as written, O(n^2), cos taken at the reduced argument (k d mod 2n).
 *   method 0: build the even extension e[m] = in[min(m, 2n-m)], m < 2n, and transform it with
 *             the radix-2 FFT (2n a power of two), keep the real part. */
static void dct1_axis(long n, long nout, const double* in, long in_stride, double* out,
                      long out_stride, int method, double* work /* >= 4*2n doubles */) {
    if (method == 1 || !is_pow2(2 * n)) {
        for (long d = 0; d < nout; ++d) {
            double acc = 0.0;
            for (long k = 0; k <= n; ++k) {
                long kd = (long)(((int64_t)k * (int64_t)d) % (int64_t)(2 * n));
                double w = (k == 0 || k == n) ? 1.0 : 2.0;
                acc += w * in[k * in_stride] * cos(ORC_PI * (double)kd / (double)n);
            }
            work[d] = acc;
        }
        for (long d = 0; d < nout; ++d) out[d * out_stride] = work[d];
    } else {
        long m2 = 2 * n;
        for (long m = 0; m < m2; ++m) {
            long k = m <= n ? m : m2 - m;
            work[2 * m] = in[k * in_stride];
            work[2 * m + 1] = 0.0;
        }
        orc_fft_radix2(m2, work, +1);
        for (long d = 0; d < nout; ++d) out[d * out_stride] = work[2 * d];
    }
}

/* Exposed for the pins: DCT-I of one vector of n+1 reals -> nout reals. */
int orc_dct1(long n, long nout, const double* in, double* out, int method) {
    if (n < 1 || nout < 1 || nout > n + 1 || !in || !out) return ORC_EINVAL;
    double* work = (double*)malloc(sizeof(double) * 8 * (size_t)(n + 1));
    if (!work) return ORC_ENOMEM;
    dct1_axis(n, nout, in, 1, out, 1, method, work);
    free(work);
    return ORC_OK;
}

/* VG, modified precompute (reading R9/R10): G_L is real and even, so of the
 * (4N)^3 samples only those at k_d in [0, 2N_d] are unique -- a (2N+1)^3 grid -- and the inverse
 * DFT above becomes, axis by axis, the DCT-I of size 2N_d+1:
 *     T[d] = 1/prod_d(4 N_d h_d) * sum_k w_kx w_ky w_kz G_L(s_k) prod_d cos(pi k_d d_d/(2 N_d)),
 * kept for 0 <= d_d <= N_d.  Memory: (2Nx+1)(2Ny+1)(2Nz+1) reals (shrinking after each axis). */
/* General form with per-axis oversampling factors m[d] (even, >= 2): the frequency lattice is
 * s_d = 2 pi k_d / (m_d N_d h_d), k_d in [0, m_d N_d / 2], and
 *     T[d] = 1/prod_d(m_d N_d h_d) * sum_k w_kx w_ky w_kz G_L(s_k) prod_d cos(2 pi k_d d_d/(m_d N_d)),
 * i.e. the DCT-I of size m_d N_d / 2 + 1 per axis.  m = (4,4,4) is the paper's choice. */
int orc_green_table_vgm(long Nx, long Ny, long Nz, const double h[3], double alpha, int method,
                        const long m[3], double* T) {
    if (Nx < 1 || Ny < 1 || Nz < 1 || !h || !T || !m || !(h[0] > 0) || !(h[1] > 0) || !(h[2] > 0) ||
        !(alpha > 0))
        return ORC_EINVAL;
    for (int d = 0; d < 3; ++d)
        if (m[d] < 2 || (m[d] & 1)) return ORC_EINVAL;
    long nx = m[0] * Nx / 2, ny = m[1] * Ny / 2, nz = m[2] * Nz / 2; /* DCT-I sizes are n+1 */
    long Kx = nx + 1, Ky = ny + 1, Kz = nz + 1;
    double L = orc_vg_window(Nx, Ny, Nz, h, alpha);
    double* f = (double*)malloc(sizeof(double) * (size_t)Kx * Ky * Kz);
    double* a = (double*)malloc(sizeof(double) * (size_t)Kx * Ky * (Nz + 1));
    double* b = (double*)malloc(sizeof(double) * (size_t)Kx * (Ny + 1) * (Nz + 1));
    if (!f || !a || !b) {
        free(f);
        free(a);
        free(b);
        return ORC_ENOMEM;
    }
#pragma omp parallel for schedule(static)
    for (long kx = 0; kx < Kx; ++kx) {
        double sx = 2.0 * ORC_PI * kx / (m[0] * Nx * h[0]);
        for (long ky = 0; ky < Ky; ++ky) {
            double sy = 2.0 * ORC_PI * ky / (m[1] * Ny * h[1]);
            for (long kz = 0; kz < Kz; ++kz) {
                double sz = 2.0 * ORC_PI * kz / (m[2] * Nz * h[2]);
                f[((size_t)kx * Ky + ky) * Kz + kz] = vg_GL(sx, sy, sz, L);
            }
        }
    }
    long nmax = nx > ny ? (nx > nz ? nx : nz) : (ny > nz ? ny : nz);
#pragma omp parallel
    {
        double* work = (double*)malloc(sizeof(double) * 8 * (size_t)(nmax + 1));
        /* axis z: f[kx][ky][kz] -> a[kx][ky][dz] */
#pragma omp for schedule(static)
        for (long p = 0; p < Kx * Ky; ++p)
            dct1_axis(nz, Nz + 1, f + (size_t)p * Kz, 1, a + (size_t)p * (Nz + 1), 1, method, work);
        /* axis y: a[kx][ky][dz] -> b[kx][dy][dz] */
#pragma omp for collapse(2) schedule(static)
        for (long kx = 0; kx < Kx; ++kx)
            for (long dz = 0; dz <= Nz; ++dz)
                dct1_axis(ny, Ny + 1, a + (size_t)kx * Ky * (Nz + 1) + dz, Nz + 1,
                          b + (size_t)kx * (Ny + 1) * (Nz + 1) + dz, Nz + 1, method, work);
        /* axis x: b[kx][dy][dz] -> T[dx][dy][dz] */
#pragma omp for schedule(static)
        for (long q = 0; q < (Ny + 1) * (Nz + 1); ++q)
            dct1_axis(nx, Nx + 1, b + q, (Ny + 1) * (Nz + 1), T + q, (Ny + 1) * (Nz + 1), method, work);
        free(work);
    }
    double scale = 1.0 / (((double)m[0] * Nx * h[0]) * ((double)m[1] * Ny * h[1]) * ((double)m[2] * Nz * h[2]));
    for (long i = 0; i < (Nx + 1) * (Ny + 1) * (Nz + 1); ++i) T[i] *= scale;
    free(f);
    free(a);
    free(b);
    return ORC_OK;
}

int orc_green_table_vg2(long Nx, long Ny, long Nz, const double h[3], double alpha, int method,
                        double* T) {
    const long m[3] = {4, 4, 4};
    return orc_green_table_vgm(Nx, Ny, Nz, h, alpha, method, m, T);
}

/* Anisotropy-safe oversampling (reading R17; SURVEY 8(c) pt 12, 8(f) N2): the kernel
 * truncated at radius L = alpha * diagonal is periodised with period m_d L_d along axis d, and
 * displacements up to L_d are used, so no image overlaps iff m_d L_d >= L + L_d.  The factors are
 * kept powers of two and never below the paper's 4:  m_d = 4, doubled while m_d < 1 + L / L_d. */
int orc_vg_safe_factors(long Nx, long Ny, long Nz, const double h[3], double alpha, long m[3]) {
    if (Nx < 1 || Ny < 1 || Nz < 1 || !h || !m || !(alpha > 0)) return ORC_EINVAL;
    double L = orc_vg_window(Nx, Ny, Nz, h, alpha);
    const long N[3] = {Nx, Ny, Nz};
    for (int d = 0; d < 3; ++d) {
        m[d] = 4;
        while ((double)m[d] < 1.0 + L / (N[d] * h[d])) m[d] *= 2;
    }
    return ORC_OK;
}

/* Step 3: G2 on the doubled grid by the 8-case mirror rule,
 * G2[i,j,k] = T[min(i,2Nx-i), min(j,2Ny-j), min(k,2Nz-k)], written as a complex array (im = 0).
 * (The index-N planes use displacement N h, R6; they cannot influence the restricted result.) */
int orc_green_g2(long Nx, long Ny, long Nz, const double* T, double* G2c) {
    if (Nx < 1 || Ny < 1 || Nz < 1 || !T || !G2c) return ORC_EINVAL;
    long Dx = 2 * Nx, Dy = 2 * Ny, Dz = 2 * Nz;
#pragma omp parallel for schedule(static)
    for (long i = 0; i < Dx; ++i) {
        long dx = i <= Nx ? i : Dx - i;
        for (long j = 0; j < Dy; ++j) {
            long dy = j <= Ny ? j : Dy - j;
            for (long k = 0; k < Dz; ++k) {
                long dz = k <= Nz ? k : Dz - k;
                size_t o = ((size_t)i * Dy + j) * Dz + k;
                G2c[2 * o] = T[(dx * (Ny + 1) + dy) * (Nz + 1) + dz];
                G2c[2 * o + 1] = 0.0;
            }
        }
    }
    return ORC_OK;
}

/* F{G2}: fills Ghat (complex, (2N)^3) = DFT3(G2).  Unscaled. */
int orc_green_spectrum(long Nx, long Ny, long Nz, const double* T, int method, double* Ghat) {
    int rc = orc_green_g2(Nx, Ny, Nz, T, Ghat);
    if (rc != ORC_OK) return rc;
    return orc_fft3d(2 * Nx, 2 * Ny, 2 * Nz, Ghat, -1, method);
}

/* Steps 1-5 of PAPER.md:67-82, literally:
 *   1-2. rho2 on the (2N)^3 grid = rho on [0,N)^3, zero elsewhere.
 *   4.   phi2 = hx hy hz F^-1{ F{rho2} x F{G2} }   (Ghat = F{G2} supplied by the caller,
 *        "reused every time step").
 *   5.   phi = phi2 restricted to [0,N)^3.
 * F^-1 carries the 1/(8 Nx Ny Nz) (R7).  eps0 = 1 (R2). */
int orc_solve(long Nx, long Ny, long Nz, const double h[3], const double* Ghat, int method,
              const double* rho, double* phi) {
    if (Nx < 1 || Ny < 1 || Nz < 1 || !h || !Ghat || !rho || !phi) return ORC_EINVAL;
    long Dx = 2 * Nx, Dy = 2 * Ny, Dz = 2 * Nz;
    size_t total = (size_t)Dx * Dy * Dz;
    double* r2 = (double*)calloc(2 * total, sizeof(double));
    if (!r2) return ORC_ENOMEM;
    for (long i = 0; i < Nx; ++i)
        for (long j = 0; j < Ny; ++j)
            for (long k = 0; k < Nz; ++k)
                r2[2 * (((size_t)i * Dy + j) * Dz + k)] = rho[((size_t)i * Ny + j) * Nz + k];
    int rc = orc_fft3d(Dx, Dy, Dz, r2, -1, method);
    if (rc != ORC_OK) {
        free(r2);
        return rc;
    }
#pragma omp parallel for schedule(static)
    for (long o = 0; o < (long)total; ++o) {
        double ar = r2[2 * o], ai = r2[2 * o + 1];
        double br = Ghat[2 * o], bi = Ghat[2 * o + 1];
        r2[2 * o] = ar * br - ai * bi;
        r2[2 * o + 1] = ar * bi + ai * br;
    }
    rc = orc_fft3d(Dx, Dy, Dz, r2, +1, method);
    if (rc != ORC_OK) {
        free(r2);
        return rc;
    }
    double scale = h[0] * h[1] * h[2] / (double)total;
    for (long i = 0; i < Nx; ++i)
        for (long j = 0; j < Ny; ++j)
            for (long k = 0; k < Nz; ++k)
                phi[((size_t)i * Ny + j) * Nz + k] = scale * r2[2 * (((size_t)i * Dy + j) * Dz + k)];
    free(r2);
    return ORC_OK;
}

/* Field output (Eq. A.1: E = -grad phi; reading R18):
 * the gradient is taken spectrally on the doubled periodic grid, where the solver already is:
 *   E_d = -hx hy hz F^-1{ i k_d F{rho2} x F{G2} } restricted,   k_d = 2 pi m'_d / (2 N_d h_d),
 *   m' = m for m < N_d, m - 2 N_d for m > N_d, and 0 at the Nyquist index m = N_d (the derivative of
 *   the real trigonometric interpolant).  phi is returned as in orc_solve.
 * E: [3][Nx][Ny][Nz] (component-major, each component laid out like phi).  phi may be NULL. */
int orc_solve_field(long Nx, long Ny, long Nz, const double h[3], const double* Ghat, int method,
                    const double* rho, double* phi, double* E) {
    if (Nx < 1 || Ny < 1 || Nz < 1 || !h || !Ghat || !rho || !E) return ORC_EINVAL;
    long D[3] = {2 * Nx, 2 * Ny, 2 * Nz};
    long Dx = D[0], Dy = D[1], Dz = D[2];
    size_t total = (size_t)Dx * Dy * Dz, V = (size_t)Nx * Ny * Nz;
    double* r2 = (double*)calloc(2 * total, sizeof(double));
    double* w2 = (double*)malloc(2 * total * sizeof(double));
    if (!r2 || !w2) { free(r2); free(w2); return ORC_ENOMEM; }
    for (long i = 0; i < Nx; ++i)
        for (long j = 0; j < Ny; ++j)
            for (long k = 0; k < Nz; ++k)
                r2[2 * (((size_t)i * Dy + j) * Dz + k)] = rho[((size_t)i * Ny + j) * Nz + k];
    int rc = orc_fft3d(Dx, Dy, Dz, r2, -1, method);
    if (rc != ORC_OK) { free(r2); free(w2); return rc; }
#pragma omp parallel for schedule(static)
    for (long o = 0; o < (long)total; ++o) {
        double ar = r2[2 * o], ai = r2[2 * o + 1];
        double br = Ghat[2 * o], bi = Ghat[2 * o + 1];
        r2[2 * o] = ar * br - ai * bi;
        r2[2 * o + 1] = ar * bi + ai * br;
    }
    double scale = h[0] * h[1] * h[2] / (double)total;
    for (int d = -1; d < 3; ++d) {   /* d = -1: phi itself */
        if (d < 0 && !phi) continue;
#pragma omp parallel for schedule(static)
        for (long i = 0; i < Dx; ++i)
            for (long j = 0; j < Dy; ++j)
                for (long k = 0; k < Dz; ++k) {
                    size_t o = ((size_t)i * Dy + j) * Dz + k;
                    double ar = r2[2 * o], ai = r2[2 * o + 1];
                    if (d < 0) { w2[2 * o] = ar; w2[2 * o + 1] = ai; continue; }
                    long m = d == 0 ? i : (d == 1 ? j : k), half = D[d] / 2;
                    long mp = m < half ? m : (m == half ? 0 : m - D[d]);
                    double kd = 2.0 * ORC_PI * (double)mp / ((double)D[d] * h[d]);
                    /* -(i kd)(ar + i ai) = kd ai - i kd ar */
                    w2[2 * o] = kd * ai;
                    w2[2 * o + 1] = -kd * ar;
                }
        rc = orc_fft3d(Dx, Dy, Dz, w2, +1, method);
        if (rc != ORC_OK) { free(r2); free(w2); return rc; }
        double* out = d < 0 ? phi : E + (size_t)d * V;
        for (long i = 0; i < Nx; ++i)
            for (long j = 0; j < Ny; ++j)
                for (long k = 0; k < Nz; ++k)
                    out[((size_t)i * Ny + j) * Nz + k] = scale * w2[2 * (((size_t)i * Dy + j) * Dz + k)];
    }
    free(r2);
    free(w2);
    return ORC_OK;
}

/* Def. O1 (PAPER.md:35 with the weight of PAPER.md:80), the plain discrete convolution:
 *   phi[i,j,k] = hx hy hz sum_{i',j',k'} T[|i-i'|,|j-j'|,|k-k'|] rho[i',j',k'].
 * Evaluated only at the npts output points listed in idx (flat C-order indices); idx == NULL
 * means all Nx Ny Nz points.  O(npts * V).
 * The V products are added in plain order in `long double` (x87 80-bit, 64-bit mantissa): the sum of
 * V ~ 1e8 terms then carries a rounding error of ~ sqrt(V) 2^-64 ~ 5e-16 instead of sqrt(V) 2^-53 ~ 1e-12,
 * so that the reference is good to the 1e-12 the GPU path is held to at the full sizes (BASELINE.json
 * north_star tolerance); only the final value is rounded to fp64. */
int orc_direct_sum(long Nx, long Ny, long Nz, const double h[3], const double* T, const double* rho,
                   long npts, const long* idx, double* out) {
    if (Nx < 1 || Ny < 1 || Nz < 1 || !h || !T || !rho || !out) return ORC_EINVAL;
    long V = Nx * Ny * Nz;
    if (!idx) npts = V;
    long double w = (long double)h[0] * (long double)h[1] * (long double)h[2];
#pragma omp parallel for schedule(dynamic, 1)
    for (long p = 0; p < npts; ++p) {
        long f = idx ? idx[p] : p;
        long i = f / (Ny * Nz), j = (f / Nz) % Ny, k = f % Nz;
        long double acc = 0.0L;
        for (long a = 0; a < Nx; ++a) {
            long dx = labs(i - a);
            for (long b = 0; b < Ny; ++b) {
                long dy = labs(j - b);
                const double* Trow = T + (dx * (Ny + 1) + dy) * (Nz + 1);
                const double* rrow = rho + ((size_t)a * Ny + b) * Nz;
                for (long c = 0; c < Nz; ++c) acc += (long double)Trow[labs(k - c)] * (long double)rrow[c];
            }
        }
        out[p] = (double)(w * acc);
    }
    return ORC_OK;
}

/* One entry of the Vico-Greengard table by the explicit triple cosine sum (G_L is real
 * and even, so the inverse DFT of PAPER.md:94-98 on the m_d N_d lattice "reduces to a discrete cosine
 * transform"; type 1), written out term by term with no transform at all:
 *     T[d] = 1/prod_d(m_d N_d h_d) * sum_{kx=0..nx} sum_{ky=0..ny} sum_{kz=0..nz}
 *                w_kx w_ky w_kz G_L(s_k) cos(pi kx dx/nx) cos(pi ky dy/ny) cos(pi kz dz/nz),
 *     n_d = m_d N_d / 2,  s_d = 2 pi k_d / (m_d N_d h_d),  w_0 = w_n = 1, w_k = 2 otherwise,
 * for the npts entries d[p] = (dx, dy, dz) listed in d (3 longs each).  m = (4,4,4) is the paper's lattice
 * (VICO / VICO_2), other even m the anisotropy-safe one (R17).  O(npts * nx ny nz): usable for a handful of
 * entries at any mesh size (the 512^3 table needs a 1025^3 lattice, 1.1e9 terms per entry), which is what the
 * full-size GPU table checks use.  The cosines are taken at arguments reduced mod 2n; sums in long double. */
int orc_green_table_vg_entries(long Nx, long Ny, long Nz, const double h[3], double alpha, const long m[3],
                               long npts, const long* d, double* out) {
    if (Nx < 1 || Ny < 1 || Nz < 1 || !h || !m || !d || !out || npts < 0 || !(h[0] > 0) || !(h[1] > 0) ||
        !(h[2] > 0) || !(alpha > 0))
        return ORC_EINVAL;
    for (int a = 0; a < 3; ++a)
        if (m[a] < 2 || (m[a] & 1)) return ORC_EINVAL;
    const long n[3] = {m[0] * Nx / 2, m[1] * Ny / 2, m[2] * Nz / 2};
    const double L = orc_vg_window(Nx, Ny, Nz, h, alpha);
    const double period[3] = {(double)m[0] * Nx * h[0], (double)m[1] * Ny * h[1], (double)m[2] * Nz * h[2]};
    int err = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (long p = 0; p < npts; ++p) {
        /* weighted cosine factors of this entry along each axis */
        double* c[3] = {NULL, NULL, NULL};
        int bad = 0;
        for (int a = 0; a < 3; ++a) {
            c[a] = (double*)malloc(sizeof(double) * (size_t)(n[a] + 1));
            if (!c[a]) { bad = 1; break; }
            for (long k = 0; k <= n[a]; ++k) {
                long kd = (long)(((int64_t)k * (int64_t)d[3 * p + a]) % (int64_t)(2 * n[a]));
                double wk = (k == 0 || k == n[a]) ? 1.0 : 2.0;
                c[a][k] = wk * cos(ORC_PI * (double)kd / (double)n[a]);
            }
        }
        if (bad) {
#pragma omp atomic write
            err = 1;
        } else {
            long double acc = 0.0L;
            for (long kx = 0; kx <= n[0]; ++kx) {
                double sx = 2.0 * ORC_PI * kx / period[0];
                long double ax = 0.0L;
                for (long ky = 0; ky <= n[1]; ++ky) {
                    double sy = 2.0 * ORC_PI * ky / period[1];
                    long double ay = 0.0L;
                    for (long kz = 0; kz <= n[2]; ++kz) {
                        double sz = 2.0 * ORC_PI * kz / period[2];
                        ay += (long double)(vg_GL(sx, sy, sz, L) * c[2][kz]);
                    }
                    ax += ay * c[1][ky];
                }
                acc += ax * c[0][kx];
            }
            out[p] = (double)(acc / ((long double)period[0] * period[1] * period[2]));
        }
        for (int a = 0; a < 3; ++a) free(c[a]);
    }
    return err ? ORC_ENOMEM : ORC_OK;
}

/* ------------------------------------------------------------------------------------------
 * Mixed periodic / open directions (PAPER.md:67 step 1: "Double the computational grid in
 * the non-periodic directions (those which have open boundary conditions)"; reading R20).
 * periodic[d] != 0: direction d is periodic with the period of the domain, L_d = N_d h_d.  The grid is NOT
 * doubled along d and rho is not padded there; step 3's "circular shifting and making G periodic"
 * along d is the nearest-image kernel G2[i] = T[min(i, N_d - i)], i < N_d.  Open directions as
 * in orc_solve: doubled, zero-padded, mirrored.  T: the (Nx+1)(Ny+1)(Nz+1) table of orc_green_table_*.
 * ------------------------------------------------------------------------------------------ */
int orc_solve_mixed(long Nx, long Ny, long Nz, const double h[3], const double* T, const int periodic[3],
                    int method, const double* rho, double* phi) {
    if (Nx < 1 || Ny < 1 || Nz < 1 || !h || !T || !periodic || !rho || !phi) return ORC_EINVAL;
    const long N[3] = {Nx, Ny, Nz};
    long D[3];
    for (int d = 0; d < 3; ++d) D[d] = periodic[d] ? N[d] : 2 * N[d];   /* step 1 */
    size_t total = (size_t)D[0] * D[1] * D[2];
    double* r2 = (double*)calloc(2 * total, sizeof(double));
    double* g2 = (double*)calloc(2 * total, sizeof(double));
    if (!r2 || !g2) { free(r2); free(g2); return ORC_ENOMEM; }
    for (long i = 0; i < Nx; ++i)                                          /* step 2 */
        for (long j = 0; j < Ny; ++j)
            for (long k = 0; k < Nz; ++k)
                r2[2 * (((size_t)i * D[1] + j) * D[2] + k)] = rho[((size_t)i * Ny + j) * Nz + k];
    for (long i = 0; i < D[0]; ++i) {                                      /* step 3 */
        long dx = i <= D[0] - i ? i : D[0] - i;   /* both cases: the distance to the nearest period of the grid */
        for (long j = 0; j < D[1]; ++j) {
            long dy = j <= D[1] - j ? j : D[1] - j;
            for (long k = 0; k < D[2]; ++k) {
                long dz = k <= D[2] - k ? k : D[2] - k;
                g2[2 * (((size_t)i * D[1] + j) * D[2] + k)] = T[(dx * (Ny + 1) + dy) * (Nz + 1) + dz];
            }
        }
    }
    int rc = orc_fft3d(D[0], D[1], D[2], r2, -1, method);                  /* step 4 */
    if (rc == ORC_OK) rc = orc_fft3d(D[0], D[1], D[2], g2, -1, method);
    if (rc == ORC_OK) {
        for (size_t o = 0; o < total; ++o) {
            double ar = r2[2 * o], ai = r2[2 * o + 1], br = g2[2 * o], bi = g2[2 * o + 1];
            r2[2 * o] = ar * br - ai * bi;
            r2[2 * o + 1] = ar * bi + ai * br;
        }
        rc = orc_fft3d(D[0], D[1], D[2], r2, +1, method);
    }
    if (rc == ORC_OK) {
        double scale = h[0] * h[1] * h[2] / (double)total;
        for (long i = 0; i < Nx; ++i)                                      /* step 5 */
            for (long j = 0; j < Ny; ++j)
                for (long k = 0; k < Nz; ++k)
                    phi[((size_t)i * Ny + j) * Nz + k] = scale * r2[2 * (((size_t)i * D[1] + j) * D[2] + k)];
    }
    free(r2);
    free(g2);
    return rc;
}

/* The same result as a plain sum (Def. O1 with the nearest image along the periodic directions):
 *   phi[i] = hx hy hz sum_j T[|i - j|*] rho[j],  |i - j|*_d = min(|i_d - j_d|, N_d - |i_d - j_d|) if d is periodic,
 *                                                             |i_d - j_d| otherwise.
 * idx / npts / long double accumulation as in orc_direct_sum. */
int orc_direct_sum_mixed(long Nx, long Ny, long Nz, const double h[3], const double* T, const int periodic[3],
                         const double* rho, long npts, const long* idx, double* out) {
    if (Nx < 1 || Ny < 1 || Nz < 1 || !h || !T || !periodic || !rho || !out) return ORC_EINVAL;
    long V = Nx * Ny * Nz;
    if (!idx) npts = V;
    long double w = (long double)h[0] * (long double)h[1] * (long double)h[2];
#pragma omp parallel for schedule(dynamic, 1)
    for (long p = 0; p < npts; ++p) {
        long f = idx ? idx[p] : p;
        long i = f / (Ny * Nz), j = (f / Nz) % Ny, k = f % Nz;
        long double acc = 0.0L;
        for (long a = 0; a < Nx; ++a) {
            long dx = labs(i - a);
            if (periodic[0] && Nx - dx < dx) dx = Nx - dx;
            for (long b = 0; b < Ny; ++b) {
                long dy = labs(j - b);
                if (periodic[1] && Ny - dy < dy) dy = Ny - dy;
                for (long c = 0; c < Nz; ++c) {
                    long dz = labs(k - c);
                    if (periodic[2] && Nz - dz < dz) dz = Nz - dz;
                    acc += (long double)T[(dx * (Ny + 1) + dy) * (Nz + 1) + dz] *
                           (long double)rho[((size_t)a * Ny + b) * Nz + c];
                }
            }
        }
        out[p] = (double)(w * acc);
    }
    return ORC_OK;
}

// green_kernels.cuh -- Green's-function precompute (done once per plan).
//
//   HE:  T[d] = 1/(4 pi |d h|), T[0] = g0.
//   VG:      G_L (Eq. 3) on the (4N)^3 lattice (stored as its C2R half spectrum), inverse DFT,
//                              restricted to d <= N.
//   VG2:    G_L on the (2N+1)^3 lattice, DCT-I per axis, restricted to d <= N.
//   all: Ghat = F{G2} of the 8-case mirror = 3-D DCT-I of T (G2 is real and even).
//
// These kernels are NOT on the per-solve path (once per plan, again when the spacing changes).  Powers of two between
// 8 and 1024 run on the warp-level transform of the solve (k_dct1_warp), other lengths on a Stockham tile kernel or the
// cosine sum as written.
#pragma once
#include <cuda_runtime.h>
#include "fft_warp.cuh"

namespace fsp {

// sin(x) up to sign for 0 <= x < 2^20 pi: x - n pi by a two-constant Cody-Waite reduction (n pi_hi is formed inside the
// fma and the difference is exactly representable, so the reduced argument carries one rounding), then the Taylor
// polynomial through x^21 on [-pi/2, pi/2] (first omitted term 1.3e-18 relative).  Eq. 3 needs sin^2 only, so the
// factor (-1)^n is never formed.  A third of the instructions of sin(): no quadrant select, no conversions, no slow path
// (the lattice argument is at most (L/2) pi sqrt(sum 1/h_d^2), 2.4e3 at 512^3; beyond the bound the library is called).
constexpr double kSinModPiMax = 3.0e6;
__device__ __forceinline__ double sin_mod_pi_nocheck(double x) {
    const double RND = 6755399441055744.0;   // 1.5 * 2^52: adding and subtracting it rounds to the nearest integer
    const double n = __dadd_rn(__fma_rn(x, 0.31830988618379067154, RND), -RND);
    double f = __fma_rn(-n, 3.141592653589793116, x);
    f = __fma_rn(-n, 1.2246467991473532e-16, f);
    const double t = f * f;
    double p = 1.0 / 51090942171709440000.0;
    p = fma(p, t, -1.0 / 121645100408832000.0);
    p = fma(p, t, 1.0 / 355687428096000.0);
    p = fma(p, t, -1.0 / 1307674368000.0);
    p = fma(p, t, 1.0 / 6227020800.0);
    p = fma(p, t, -1.0 / 39916800.0);
    p = fma(p, t, 1.0 / 362880.0);
    p = fma(p, t, -1.0 / 5040.0);
    p = fma(p, t, 1.0 / 120.0);
    p = fma(p, t, -1.0 / 6.0);
    return fma(f * t, p, f);
}
__device__ __forceinline__ double sin_mod_pi(double x) { return x > kSinModPiMax ? sin(x) : sin_mod_pi_nocheck(x); }

// Eq. 3 with the s -> 0 limit L^2/2.
// (1/|s| by rsqrt: one reciprocal square root instead of a square root and a division -- the fill is evaluated inside
// the first DCT pass, 1.1e9 lattice points at 512^3, and is bound by fp64 instructions)
__device__ __forceinline__ double vg_GL(double sx, double sy, double sz, double L) {
    const double s2 = sx * sx + sy * sy + sz * sz;
    if (s2 == 0.0) return 0.5 * L * L;
    const double r = rsqrt(s2);
    const double q = sin_mod_pi(0.5 * L * (s2 * r)) * r;
    return 2.0 * q * q;
}
// 1/sqrt(x) without the special-case branch of rsqrt() (whose slow-path call splits every evaluation into basic blocks
// of its own and keeps independent evaluations from interleaving): fp32 seed, two Newton steps in fp64 (relative error
// 1e-7 -> 1.5e-14 -> 3e-28, i.e. the rounding of the last step).  x in [kRsqrtMin, kRsqrtMax] (the fp32 range).
constexpr double kRsqrtMin = 1.0e-35, kRsqrtMax = 1.0e37;
__device__ __forceinline__ double rsqrt_straight(double x) {
    const double y0 = (double)rsqrtf((float)x);
    const double hx = 0.5 * x;
    double e = fma(-hx * y0, y0, 0.5);
    const double y1 = fma(y0, e, y0);
    e = fma(-hx * y1, y1, 0.5);
    return fma(y1, e, y1);
}
// Eq. 3 without a branch, for arguments known to stay below kSinModPiMax and s^2 inside the range of rsqrt_straight or
// zero (the caller checks its pencil): independent evaluations then interleave in one instruction stream.  s = 0: s^2 is
// raised to kRsqrtMin, where sin(x) = x to the last bit and the formula returns its own limit 2 (L/2)^2.
__device__ __forceinline__ double vg_GL_straight(double s2xy, double sz, double halfL) {
    const double s2 = fmax(fma(sz, sz, s2xy), kRsqrtMin);
    const double r = rsqrt_straight(s2);
    const double q = sin_mod_pi_nocheck(halfL * (s2 * r)) * r;
    return 2.0 * q * q;
}

// Periodic directions (R20): along a periodic direction d the kernel is made
// periodic with the period of the domain, T'[i] = T[min(i, N_d - i)], i <= N_d.  Its mirror image on the doubled grid
// (what the DCT-I below transforms) is then exactly the N_d-periodic repetition of the nearest-image kernel, whose
// 2 N_d-point spectrum has zero odd bins: the five solve kernels, unchanged, compute the CYCLIC convolution of period
// N_d along d and the free-space one along the others.  In place: an entry is rewritten only if one of its indices
// folds, and the entries it is copied from (all indices <= N_d / 2 along the periodic directions) never are.
__global__ void k_fold_periodic(double* __restrict__ T, int Nx, int Ny, int Nz, int mask) {
    const long total = (long)(Nx + 1) * (Ny + 1) * (Nz + 1);
    for (long o = blockIdx.x * (long)blockDim.x + threadIdx.x; o < total; o += (long)gridDim.x * blockDim.x) {
        const int dz = (int)(o % (Nz + 1));
        const int dy = (int)((o / (Nz + 1)) % (Ny + 1));
        const int dx = (int)(o / ((long)(Nz + 1) * (Ny + 1)));
        const int fx = (mask & 1) && Nx - dx < dx ? Nx - dx : dx;
        const int fy = (mask & 2) && Ny - dy < dy ? Ny - dy : dy;
        const int fz = (mask & 4) && Nz - dz < dz ? Nz - dz : dz;
        if (fx != dx || fy != dy || fz != dz) T[o] = T[((long)fx * (Ny + 1) + fy) * (Nz + 1) + fz];
    }
}

__global__ void k_fill_he(double* __restrict__ T, int Nx, int Ny, int Nz, double hx, double hy,
                          double hz, double g0) {
    const long total = (long)(Nx + 1) * (Ny + 1) * (Nz + 1);
    for (long o = blockIdx.x * (long)blockDim.x + threadIdx.x; o < total; o += (long)gridDim.x * blockDim.x) {
        const int dz = (int)(o % (Nz + 1));
        const int dy = (int)((o / (Nz + 1)) % (Ny + 1));
        const int dx = (int)(o / ((long)(Nz + 1) * (Ny + 1)));
        const double x = dx * hx, y = dy * hy, z = dz * hz;
        const double r = sqrt(x * x + y * y + z * z);
        T[o] = (o == 0) ? g0 : 1.0 / (4.0 * 3.14159265358979323846 * r);
    }
}

// VG2 / VG-safe: f[kx][ky][kz] = G_L(2 pi k_d / (m_d N_d h_d)), 0 <= k_d <= m_d N_d / 2
// (m = 4 on every axis is the paper's lattice; R17 for the per-axis factors)
__global__ void k_fill_gl_vg2(double* __restrict__ f, int Nx, int Ny, int Nz, double hx, double hy,
                              double hz, double L, int mx, int my, int mz) {
    const long Kx = (long)mx * Nx / 2 + 1, Ky = (long)my * Ny / 2 + 1, Kz = (long)mz * Nz / 2 + 1;
    const long total = Kx * Ky * Kz;
    const double PI2 = 6.28318530717958647692;
    for (long o = blockIdx.x * (long)blockDim.x + threadIdx.x; o < total; o += (long)gridDim.x * blockDim.x) {
        const long kz = o % Kz, ky = (o / Kz) % Ky, kx = o / (Kz * Ky);
        f[o] = vg_GL(PI2 * kx / ((double)mx * Nx * hx), PI2 * ky / ((double)my * Ny * hy),
                     PI2 * kz / ((double)mz * Nz * hz), L);
    }
}

// VG (plain): the (4N)^3 lattice of G_L is real, so its inverse DFT is a C2R transform and only
// the half spectrum kx in [0, 2Nx] is stored: g[kx][iy][iz] complex, (2Nx+1) x 4Ny x 4Nz, ky and kz in DFT
// frequency order {0..2N-1, -2N..-1} (513 x 1024 x 1024 complex = 8.6 GB at 256^3).
__global__ void k_fill_gl_vg_half(double2* __restrict__ g, int Nx, int Ny, int Nz, double hx, double hy,
                                  double hz, double L) {
    const long Kx = 2L * Nx + 1, My = 4L * Ny, Mz = 4L * Nz;
    const long total = Kx * My * Mz;
    const double PI2 = 6.28318530717958647692;
    for (long o = blockIdx.x * (long)blockDim.x + threadIdx.x; o < total; o += (long)gridDim.x * blockDim.x) {
        const long iz = o % Mz, iy = (o / Mz) % My, kx = o / (Mz * My);
        const long ky = iy < 2 * Ny ? iy : iy - My, kz = iz < 2 * Nz ? iz : iz - Mz;
        g[o] = make_double2(vg_GL(PI2 * kx / (4.0 * Nx * hx), PI2 * ky / (My * hy), PI2 * kz / (Mz * hz), L), 0.0);
    }
}

// Radix-2 Stockham FFT of length Lf (power of two) in shared memory, all threads of the CTA.
// a holds the input; a and b ping-pong; returns the buffer holding the (natural-order) result.
// sign = -1 forward, +1 inverse (unscaled).
__device__ __forceinline__ double2* smem_fft_radix2(double2* a, double2* b, int Lf, int sign) {
    const int half = Lf >> 1;
    for (int Ns = 1; Ns < Lf; Ns <<= 1) {
        __syncthreads();
        for (int j = threadIdx.x; j < half; j += blockDim.x) {
            const int k = j & (Ns - 1);
            double s, c;
            sincospi((double)sign * (double)k / (double)Ns, &s, &c);  // exp(sign * 2 pi i k / (2 Ns))
            const double2 u = a[j], v0 = a[j + half];
            const double2 v = make_double2(v0.x * c - v0.y * s, v0.x * s + v0.y * c);
            const int j0 = ((j - k) << 1) + k;
            b[j0] = make_double2(u.x + v.x, u.y + v.y);
            b[j0 + Ns] = make_double2(u.x - v.x, u.y - v.y);
        }
        double2* tmp = a; a = b; b = tmp;
    }
    __syncthreads();
    return a;
}

// Un-normalised DCT-I (REDFT00) of pencils: n+1 real inputs -> first nout outputs,
//   out[d] = sum_k w_k in[k] cos(pi k d / n),  w_0 = w_n = 1, else 2,
// evaluated as the length-2n DFT of the even extension.
__global__ void k_dct1_pencils(const double* __restrict__ in, double* __restrict__ out, int n, int nout,
                               long sa_in, long sa_out, long n2, long s1_in, long s2_in, long s1_out,
                               long s2_out, double scale) {
    extern __shared__ double2 sm[];
    const int Lf = 2 * n;
    double2* a = sm;
    double2* b = sm + Lf;
    const long p = blockIdx.x;
    const double* src = in + (p / n2) * s1_in + (p % n2) * s2_in;
    double* dst = out + (p / n2) * s1_out + (p % n2) * s2_out;
    for (int m = threadIdx.x; m < Lf; m += blockDim.x) {
        const int k = m <= n ? m : Lf - m;
        a[m] = make_double2(src[(long)k * sa_in], 0.0);
    }
    double2* r = smem_fft_radix2(a, b, Lf, +1);
    for (int d = threadIdx.x; d < nout; d += blockDim.x) dst[(long)d * sa_out] = scale * r[d].x;
}

// Stockham autosort FFT of S sequences of Lf complex points held in shared memory (sequence q at a + q*Lf), all
// threads of the CTA: radix-4 stages (half the exchanges and barriers of radix 2), then one radix-2 stage if
// log2(Lf) is odd.  Sign +: exp(+2 pi i ..), i.e. the unscaled inverse DFT.  tw[k] = exp(+2 pi i k / Lf), k < Lf/2.
// a and b ping-pong; returns the buffer that holds the natural-order result (a barrier has been passed).
__device__ __forceinline__ double2* smem_stockham(double2* a, double2* b, const double2* __restrict__ tw, int S, int Lf) {
    const int half = Lf >> 1;
    int Ns = 1;
    const int quarter = Lf >> 2;
    for (; Ns * 4 <= Lf; Ns <<= 2) {
        __syncthreads();
        const int tstep = quarter / Ns;   // w1 = exp(2 pi i k / (4 Ns)) = tw[k * Lf / (4 Ns)]
        for (int e = threadIdx.x; e < S * quarter; e += blockDim.x) {
            const int q = e / quarter, j = e - q * quarter;
            const int k = j & (Ns - 1);
            const double2 w1 = tw[k * tstep], w2 = tw[2 * k * tstep];
            const double2 w3 = make_double2(w1.x * w2.x - w1.y * w2.y, w1.x * w2.y + w1.y * w2.x);
            const double2* aq = a + (long)q * Lf;
            double2* bq = b + (long)q * Lf;
            const double2 x0 = aq[j], y1 = aq[j + quarter], y2 = aq[j + 2 * quarter], y3 = aq[j + 3 * quarter];
            const double2 x1 = make_double2(y1.x * w1.x - y1.y * w1.y, y1.x * w1.y + y1.y * w1.x);
            const double2 x2 = make_double2(y2.x * w2.x - y2.y * w2.y, y2.x * w2.y + y2.y * w2.x);
            const double2 x3 = make_double2(y3.x * w3.x - y3.y * w3.y, y3.x * w3.y + y3.y * w3.x);
            const double2 s02 = make_double2(x0.x + x2.x, x0.y + x2.y), d02 = make_double2(x0.x - x2.x, x0.y - x2.y);
            const double2 s13 = make_double2(x1.x + x3.x, x1.y + x3.y), d13 = make_double2(x1.x - x3.x, x1.y - x3.y);
            const int j0 = ((j - k) << 2) + k;
            bq[j0] = make_double2(s02.x + s13.x, s02.y + s13.y);
            bq[j0 + Ns] = make_double2(d02.x - d13.y, d02.y + d13.x);          // + i (x1 - x3)
            bq[j0 + 2 * Ns] = make_double2(s02.x - s13.x, s02.y - s13.y);
            bq[j0 + 3 * Ns] = make_double2(d02.x + d13.y, d02.y - d13.x);      // - i (x1 - x3)
        }
        double2* t2 = a; a = b; b = t2;
    }
    for (; Ns < Lf; Ns <<= 1) {
        __syncthreads();
        const int tstep = half / Ns;
        for (int e = threadIdx.x; e < S * half; e += blockDim.x) {
            const int q = e / half, j = e - q * half;
            const int k = j & (Ns - 1);
            const double2 w = tw[k * tstep];
            const double2* aq = a + (long)q * Lf;
            double2* bq = b + (long)q * Lf;
            const double2 u = aq[j], v0 = aq[j + half];
            const double2 v = make_double2(v0.x * w.x - v0.y * w.y, v0.x * w.y + v0.y * w.x);
            const int j0 = ((j - k) << 1) + k;
            bq[j0] = make_double2(u.x + v.x, u.y + v.y);
            bq[j0 + Ns] = make_double2(u.x - v.x, u.y - v.y);
        }
        double2* t2 = a; a = b; b = t2;
    }
    __syncthreads();
    return a;
}

// The same DCT-I for a TILE of C adjacent pencils per CTA (C even): pencils (a, b0 .. b0+C-1) of an
// nA x nB pencil grid; element k of pencil (a, b) at in[a*sA + b*sB + k*sK].  Two things make it several
// times faster than k_dct1_pencils: (1) two real-even pencils are packed as the real and imaginary part of
// ONE complex sequence -- both transforms are real, so they come out as Re and Im of the result; (2) the
// tile is chosen along the contiguous dimension, so that global accesses are full sectors; the twiddles
// come from a shared-memory table filled once per CTA.  Shared memory: [tw: Lf/2][a: C/2*Lf][b: C/2*Lf].
// FILL: the input is not read but evaluated in place, element k of pencil (a, b) = G_L(gl.sa (gl.a0 + a), gl.sb b,
// gl.sk k) (first pass of the modified Vico-Greengard precompute: the (2N+1)^3 lattice of PAPER.md:100-102 is never
// written to memory).
struct GLFill { double sa, sb, sk, L; long a0; };
template <int C, bool FILL = false>
__global__ void k_dct1_tile(const double* __restrict__ in, double* __restrict__ out, int n, int nout,
                            long nB, long sA_in, long sB_in, long sK_in, long sA_out, long sB_out,
                            long sK_out, double scale, const GLFill gl) {
    extern __shared__ double2 sm[];
    const int Lf = 2 * n, half = n, S = C / 2;
    double2* tw = sm;
    double2* a = sm + half;
    double2* b = a + (long)S * Lf;
    const long tilesB = (nB + C - 1) / C;
    const long ia = blockIdx.x / tilesB, b0 = (blockIdx.x % tilesB) * C;
    const int nc = (int)(nB - b0 < C ? nB - b0 : C);   // pencils of this tile
    const double* src = in + ia * sA_in + b0 * sB_in;
    double* dst = out + ia * sA_out + b0 * sB_out;
    for (int k = threadIdx.x; k < half; k += blockDim.x) {
        double sn, cs;
        sincospi((double)k / (double)half, &sn, &cs);   // exp(+2 pi i k / Lf)
        tw[k] = make_double2(cs, sn);
    }
    double* af = reinterpret_cast<double*>(a);
    // load with the even extension: position m and Lf - m both hold input k
    const int total = (n + 1) * C;
    for (int e = threadIdx.x; e < total; e += blockDim.x) {
        int k, c;
        if (sK_in == 1) { k = e % (n + 1); c = e / (n + 1); }   // contiguous transform axis: k fastest
        else { c = e % C; k = e / C; }                          // strided axis: pencils fastest
        double v = 0.0;
        if (c < nc) {
            if constexpr (FILL) v = vg_GL(gl.sa * (double)(gl.a0 + ia), gl.sb * (double)(b0 + c), gl.sk * (double)k, gl.L);
            else v = src[(long)c * sB_in + (long)k * sK_in];
        }
        const long sq = (long)(c >> 1) * Lf;
        af[2 * (sq + k) + (c & 1)] = v;
        if (k > 0 && k < n) af[2 * (sq + Lf - k) + (c & 1)] = v;
    }
    a = smem_stockham(a, b, tw, S, Lf);
    const double* rf = reinterpret_cast<const double*>(a);
    const int ototal = nout * C;
    for (int e = threadIdx.x; e < ototal; e += blockDim.x) {
        int d, c;
        if (sK_out == 1) { d = e % nout; c = e / nout; }
        else { c = e % C; d = e / C; }
        if (c < nc) dst[(long)c * sB_out + (long)d * sK_out] = scale * rf[2 * ((long)(c >> 1) * Lf + d) + (c & 1)];
    }
}

// DCT-I of pencils whose length is not a power of two (meshes 3 * 2^k, 5 * 2^k): the cosine sum as
// written, out[d] = sum_k w_k in[k] cos(pi k d / n), O(n * nout) per pencil -- a once-per-plan step on meshes the
// paper never uses; the cosines come from a shared-memory table cos(pi m / n), m < 2n, indexed by (k d) mod 2n.
// Same tile geometry and FILL option as k_dct1_tile; shared memory: [table: 2n doubles][input: (n+1) * C doubles].
template <int C, bool FILL = false>
__global__ void k_dct1_direct(const double* __restrict__ in, double* __restrict__ out, int n, int nout, long nB,
                              long sA_in, long sB_in, long sK_in, long sA_out, long sB_out, long sK_out,
                              double scale, const GLFill gl) {
    extern __shared__ double smd[];
    double* ct = smd;               // 2n
    double* x = smd + 2 * n;        // (n + 1) * C, [k][c]
    const long tilesB = (nB + C - 1) / C;
    const long ia = blockIdx.x / tilesB, b0 = (blockIdx.x % tilesB) * C;
    const int nc = (int)(nB - b0 < C ? nB - b0 : C);
    const double* src = in + ia * sA_in + b0 * sB_in;
    double* dst = out + ia * sA_out + b0 * sB_out;
    for (int m = threadIdx.x; m < 2 * n; m += blockDim.x) ct[m] = cospi((double)m / (double)n);
    const int total = (n + 1) * C;
    for (int e = threadIdx.x; e < total; e += blockDim.x) {
        int k, c;
        if (sK_in == 1) { k = e % (n + 1); c = e / (n + 1); }
        else { c = e % C; k = e / C; }
        double v = 0.0;
        if (c < nc) {
            if constexpr (FILL) v = vg_GL(gl.sa * (double)(gl.a0 + ia), gl.sb * (double)(b0 + c), gl.sk * (double)k, gl.L);
            else v = src[(long)c * sB_in + (long)k * sK_in];
        }
        x[k * C + c] = (k == 0 || k == n) ? v : 2.0 * v;   // endpoint weight 1, interior weight 2
    }
    __syncthreads();
    const int ototal = nout * C;
    for (int e = threadIdx.x; e < ototal; e += blockDim.x) {
        int d, c;
        if (sK_out == 1) { d = e % nout; c = e / nout; }
        else { c = e % C; d = e / C; }
        double acc = 0.0;
        int idx = 0;   // (k d) mod 2n
        for (int k = 0; k <= n; ++k) {
            acc = fma(x[k * C + c], ct[idx], acc);
            idx += d;
            if (idx >= 2 * n) idx -= 2 * n;
        }
        if (c < nc) dst[(long)c * sB_out + (long)d * sK_out] = scale * acc;
    }
}

// DCT-I of pencils on the warp-level transform of the solve (n = M a power of two, 8 <= M <= 1024): the even extension
// e[m], m < 2M, of the pencil is REAL, so its DFT is that of the complex sequence z[j] = e[2j] + i e[2j+1], j < M,
// untangled:  X[d] = Re FFT_2M(e)[d] = 1/2 (Zr[d] + Zr[p] - s_d (Zr[d] - Zr[p]) + c_d (Zi[d] + Zi[p])),  p = (M - d) mod M,
// (c_d, s_d) = (cos, sin)(pi d / M).  One pencil per lane group of Fft2Cfg<M> (T lanes, R points per lane, lane-constant
// stage-2 twiddles, one private exchange): the partner Z[p] sits in lane T - t at register R - 1 - i (lane 0: its own
// register R - i), i.e. one shuffle per value.  Replaces the radix-4 Stockham tile kernel (six trips of every sequence
// through shared memory with CTA barriers) at these lengths: 10 x fewer cycles per pencil.  Persistent warps.
// roots: exp(-2 pi i m / 2M), m <= M (host table); lane_g: make_lane_table(M).
template <int M, bool FILL = false>
__global__ void __launch_bounds__(256, 1)
k_dct1_warp(const double* __restrict__ in, double* __restrict__ out, int nout, long nA, long nB, long sA_in, long sB_in,
            long sK_in, long sA_out, long sB_out, long sK_out, double scale, const GLFill gl,
            const double* __restrict__ lane_g, const double2* __restrict__ roots) {
    using Cfg = Fft2Cfg<M>;
    constexpr int R = Cfg::R, T = Cfg::T, G = 32 / T, NC = LaneTw<Cfg::R2>::NC, NB2 = Cfg::NB2, WARPS = 8;
    extern __shared__ double2 smw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane / T, t = lane % T;
    double2* buf = smw + (warp * G + g) * Cfg::BUF;
    double cc[NB2][NC], tn[NB2][NC];
#pragma unroll
    for (int m = 0; m < NB2; ++m)
#pragma unroll
        for (int i = 0; i < NC; ++i) {
            cc[m][i] = lane_g[(t + T * m) * 2 * NC + i];
            tn[m][i] = lane_g[(t + T * m) * 2 * NC + NC + i];
        }
    const long npencils = nA * nB;
    const long ngroups = (npencils + G - 1) / G;
    for (long grp = (long)blockIdx.x * WARPS + warp; grp < ngroups; grp += (long)gridDim.x * WARPS) {
        const long q = grp * G + g;
        const bool valid = q < npencils;
        const long ia = valid ? q / nB : 0, ib = valid ? q % nB : 0;
        const double* src = in + ia * sA_in + ib * sB_in;
        double* dst = out + ia * sA_out + ib * sB_out;
        double zr[R], zi[R];
        if constexpr (FILL) {   // every lattice value once (each enters the even extension twice): through the exchange buffer
            double* xs = reinterpret_cast<double*>(buf);
            __syncwarp();   // the previous pencil's exchange has been read back
            const double sxv = gl.sa * (double)(gl.a0 + ia), syv = gl.sb * (double)ib, s2xy = sxv * sxv + syv * syv;
            const double szmax = gl.sk * (double)M, halfL = 0.5 * gl.L;
            const double s2max = fma(szmax, szmax, s2xy);
            // (uniform over the lane group) arguments in the range of the branch-free forms: sin below its bound, every
            // non-zero s^2 of the pencil inside the fp32 range of the rsqrt seed
            if (halfL * sqrt(s2max) < kSinModPiMax && s2max < kRsqrtMax && gl.sk * gl.sk > kRsqrtMin &&
                (s2xy == 0.0 || s2xy > kRsqrtMin)) {
                // M / T full rounds with a compile-time trip count (no bound check, no branch: the evaluations of a
                // lane interleave, eight sin / rsqrt chains in flight), then the one entry k = M
#pragma unroll 8
                for (int i = 0; i < M / T; ++i) xs[t + T * i] = vg_GL_straight(s2xy, gl.sk * (double)(t + T * i), halfL);
                const double last = vg_GL_straight(s2xy, szmax, halfL);
                if (t == 0) xs[M] = last;
            } else {
                for (int k = t; k <= M; k += T) xs[k] = vg_GL(sxv, syv, gl.sk * (double)k, gl.L);
            }
            __syncwarp();
        }
#pragma unroll
        for (int i = 0; i < R; ++i) {   // z[j] = e[2j] + i e[2j+1], e[m] = x[min(m, 2M - m)]
            const int j = t + T * i;
            const int k0 = 2 * j <= M ? 2 * j : 2 * M - 2 * j, k1 = 2 * j + 1 <= M ? 2 * j + 1 : 2 * M - 2 * j - 1;
            if constexpr (FILL) {
                const double* xs = reinterpret_cast<const double*>(buf);
                zr[i] = xs[k0];
                zi[i] = xs[k1];
            } else {
                zr[i] = valid ? src[(long)k0 * sK_in] : 0.0;
                zi[i] = valid ? src[(long)k1 * sK_in] : 0.0;
            }
        }
        fft2_forward_lc<Cfg>(zr, zi, t, buf, cc, tn);
        const int pl = (T - t) % T + g * T;   // lane that holds Z[M - d] for this lane's d (lane 0 of the group: itself)
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const int d = t + T * i;
            // partner register: R - 1 - i in lane T - t; for t = 0 the lane's own register (R - i) mod R
            const double pr_s = __shfl_sync(0xffffffffu, zr[R - 1 - i], pl), pi_s = __shfl_sync(0xffffffffu, zi[R - 1 - i], pl);
            const double pr = t == 0 ? zr[(R - i) % R] : pr_s, pi = t == 0 ? zi[(R - i) % R] : pi_s;
            if (T * i < nout) {   // (uniform per register; lanes beyond nout are masked at the store)
                const double2 w = roots[d];   // (cos, -sin)(pi d / M)
                const double x = 0.5 * (zr[i] + pr + w.y * (zr[i] - pr) + w.x * (zi[i] + pi));
                if (valid && d < nout) dst[(long)d * sK_out] = scale * x;
            }
        }
        if (valid && t == 0 && M < nout) dst[(long)M * sK_out] = scale * (zr[0] - zi[0]);   // d = M: Z[M] = Z[0], c = -1, s = 0
    }
}

// Unscaled inverse complex DFT (sign +) of length Lf along one axis for a TILE of C adjacent pencils per CTA, in
// place or out of place (plain VG, y and z axes of the half-spectrum lattice).  Same tiling as k_dct1_tile: the C
// pencils are adjacent along the contiguous dimension, so the strided axes are read and written in full sectors
// (C x 16 bytes per row); element k of pencil (a, b) at data[a*sA + b*sB + k*sK].  Only pencils b < nB are
// transformed (the later passes need the columns d <= N only).  Shared memory: [tw: Lf/2][a: C*Lf][b: C*Lf].
template <int C>
__global__ void k_ifft_tile(double2* __restrict__ data, int Lf, long nB, long sA, long sB, long sK) {
    extern __shared__ double2 sm[];
    const int half = Lf >> 1;
    double2* tw = sm;
    double2* a = sm + half;
    double2* b = a + (long)C * Lf;
    const long tilesB = (nB + C - 1) / C;
    const long ia = blockIdx.x / tilesB, b0 = (blockIdx.x % tilesB) * C;
    const int nc = (int)(nB - b0 < C ? nB - b0 : C);
    double2* base = data + ia * sA + b0 * sB;
    for (int k = threadIdx.x; k < half; k += blockDim.x) {
        double sn, cs;
        sincospi((double)k / (double)half, &sn, &cs);   // exp(+2 pi i k / Lf)
        tw[k] = make_double2(cs, sn);
    }
    const int total = Lf * C;
    for (int e = threadIdx.x; e < total; e += blockDim.x) {
        int k, c;
        if (sK == 1) { k = e % Lf; c = e / Lf; }
        else { c = e % C; k = e / C; }
        a[(long)c * Lf + k] = c < nc ? base[(long)c * sB + (long)k * sK] : make_double2(0.0, 0.0);
    }
    a = smem_stockham(a, b, tw, C, Lf);
    for (int e = threadIdx.x; e < total; e += blockDim.x) {
        int k, c;
        if (sK == 1) { k = e % Lf; c = e / Lf; }
        else { c = e % C; k = e / C; }
        if (c < nc) base[(long)c * sB + (long)k * sK] = a[(long)c * Lf + k];
    }
}

// C2R along one axis for a tile of C adjacent pencils (C even): the input holds the half spectrum X[k], k <= Lf/2,
// of a REAL sequence of length Lf (X[Lf-k] = conj X[k]); outputs x[n] = sum_k X[k] exp(+2 pi i k n / Lf), n < nout,
// times `scale`.  Two real transforms per complex FFT: pencils 2q and 2q+1 are packed as Z = A + i B (with the
// Hermitian extension Z[Lf-k] = conj A[k] + i conj B[k]), and come out as Re z and Im z.  Last pass of the plain VG
// precompute: in = the lattice after its y and z passes, out = the table T (restriction to n <= N).
template <int C>
__global__ void k_c2r_tile(const double2* __restrict__ in, double* __restrict__ out, int Lf, int nout, long nB,
                           long sA_in, long sB_in, long sK_in, long sA_out, long sB_out, long sK_out, double scale) {
    extern __shared__ double2 sm[];
    const int half = Lf >> 1, S = C / 2;
    double2* tw = sm;
    double2* a = sm + half;
    double2* b = a + (long)S * Lf;
    const long tilesB = (nB + C - 1) / C;
    const long ia = blockIdx.x / tilesB, b0 = (blockIdx.x % tilesB) * C;
    const int nc = (int)(nB - b0 < C ? nB - b0 : C);
    const double2* src = in + ia * sA_in + b0 * sB_in;
    double* dst = out + ia * sA_out + b0 * sB_out;
    for (int k = threadIdx.x; k < half; k += blockDim.x) {
        double sn, cs;
        sincospi((double)k / (double)half, &sn, &cs);
        tw[k] = make_double2(cs, sn);
    }
    const int total = (half + 1) * S;
    for (int e = threadIdx.x; e < total; e += blockDim.x) {
        int k, q;
        if (sK_in == 1) { k = e % (half + 1); q = e / (half + 1); }
        else { q = e % S; k = e / S; }
        const int c0 = 2 * q, c1 = 2 * q + 1;
        const double2 A = c0 < nc ? src[(long)c0 * sB_in + (long)k * sK_in] : make_double2(0.0, 0.0);
        const double2 B = c1 < nc ? src[(long)c1 * sB_in + (long)k * sK_in] : make_double2(0.0, 0.0);
        a[(long)q * Lf + k] = make_double2(A.x - B.y, A.y + B.x);                       // A + i B
        if (k > 0 && k < half) a[(long)q * Lf + Lf - k] = make_double2(A.x + B.y, B.x - A.y);   // conj A + i conj B
    }
    a = smem_stockham(a, b, tw, S, Lf);
    const double* rf = reinterpret_cast<const double*>(a);
    const int ototal = nout * C;
    for (int e = threadIdx.x; e < ototal; e += blockDim.x) {
        int d, c;
        if (sK_out == 1) { d = e % nout; c = e / nout; }
        else { c = e % C; d = e / C; }
        if (c < nc) dst[(long)c * sB_out + (long)d * sK_out] = scale * rf[2 * ((long)(c >> 1) * Lf + d) + (c & 1)];
    }
}

// Spectrum layout for K3 (k_conv_z_p, k_conv_z_w): the unique octant only, rows de-interleaved by parity of kz:
//   Gk[(kx*(Ny+1) + qy)*(Nz+2) + m]              = scale * Goct[kx][qy][2m],    m <= Nz/2   (E)
//   Gk[(kx*(Ny+1) + qy)*(Nz+2) + Nz/2 + 1 + m]   = scale * Goct[kx][qy][2m+1],  m <  Nz/2   (O)
__global__ void k_layout_spectrum_oct(const double* __restrict__ Goct, double* __restrict__ Gk, int Nx,
                                      int Ny, int Nz, double scale) {
    const long row = Nz + 2;
    const long total = (long)(Nx + 1) * (Ny + 1) * row;
    for (long o = blockIdx.x * (long)blockDim.x + threadIdx.x; o < total; o += (long)gridDim.x * blockDim.x) {
        const int c = (int)(o % row);
        const long pr = o / row;
        double v = 0.0;
        if (c <= Nz / 2) v = Goct[pr * (Nz + 1) + 2 * c];
        else if (c <= Nz) v = Goct[pr * (Nz + 1) + 2 * (c - Nz / 2 - 1) + 1];
        Gk[o] = scale * v;
    }
}

// Spectrum layout for k_conv_z_f: the unique octant, rows in natural order with one pad element:
//   Gk[(kx*(Ny+1) + qy)*(Nz+2) + kz] = scale * Goct[kx][qy][kz],  kz <= Nz
__global__ void k_layout_spectrum_nat(const double* __restrict__ Goct, double* __restrict__ Gk, int Nx,
                                      int Ny, int Nz, double scale) {
    const long row = Nz + 2;
    const long total = (long)(Nx + 1) * (Ny + 1) * row;
    for (long o = blockIdx.x * (long)blockDim.x + threadIdx.x; o < total; o += (long)gridDim.x * blockDim.x) {
        const int c = (int)(o % row);
        const long pr = o / row;
        Gk[o] = c <= Nz ? scale * Goct[pr * (Nz + 1) + c] : 0.0;
    }
}

// Spectrum layout for k_conv_z_pf (Nz = 3 P / 2): all M2 = 2 Nz = 3 P entries of a row in CRT order,
//   Gk[row * M2 + k1 * P + k2] = scale * Goct[row][min(k, M2 - k)],   k = k1 (mod 3), k = k2 (mod P)
__global__ void k_layout_spectrum_pfa(const double* __restrict__ Goct, double* __restrict__ Gk, int Nx, int Ny,
                                      int Nz, int P, int c1, int c2, double scale) {
    const long row = 2L * Nz;
    const long total = (long)(Nx + 1) * (Ny + 1) * row;
    for (long o = blockIdx.x * (long)blockDim.x + threadIdx.x; o < total; o += (long)gridDim.x * blockDim.x) {
        const int c = (int)(o % row);
        const long pr = o / row;
        const int k1 = c / P, k2 = c % P;
        const int k = (int)(((long)c1 * k1 + (long)c2 * k2) % row);
        const int idx = k <= Nz ? k : (int)row - k;
        Gk[o] = scale * Goct[pr * (Nz + 1) + idx];
    }
}

}  // namespace fsp

// green_kernels.cuh -- Green's-function precompute (done once per plan).
//
//   HE:  T[d] = 1/(4 pi |d h|), T[0] = g0.
//   VG:      G_L (Eq. 3) on the (4N)^3 lattice, inverse DFT, restricted to d <= N.
//   VG2:    G_L on the (2N+1)^3 lattice, DCT-I per axis, restricted to d <= N.
//   all: Ghat = F{G2} of the 8-case mirror = 3-D DCT-I of T (G2 is real and even).
//
// These kernels are NOT on the per-solve path and are written for clarity, not speed: one CTA
// transforms one pencil with a radix-2 Stockham FFT in shared memory; twiddles come from
// sincospi() in fp64.
#pragma once
#include <cuda_runtime.h>

namespace fsp {

// Eq. 3 with the s -> 0 limit L^2/2.
__device__ __forceinline__ double vg_GL(double sx, double sy, double sz, double L) {
    const double s = sqrt(sx * sx + sy * sy + sz * sz);
    if (s == 0.0) return 0.5 * L * L;
    const double q = sin(0.5 * L * s) / s;
    return 2.0 * q * q;
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

// VG: g[ix][iy][iz] complex on the (4N)^3 lattice, DFT frequency order k in {0..2N-1, -2N..-1}
__global__ void k_fill_gl_vg(double2* __restrict__ g, int Nx, int Ny, int Nz, double hx, double hy,
                             double hz, double L) {
    const long Mx = 4 * Nx, My = 4 * Ny, Mz = 4 * Nz;
    const long total = Mx * My * Mz;
    const double PI2 = 6.28318530717958647692;
    for (long o = blockIdx.x * (long)blockDim.x + threadIdx.x; o < total; o += (long)gridDim.x * blockDim.x) {
        const long iz = o % Mz, iy = (o / Mz) % My, ix = o / (Mz * My);
        const long kx = ix < 2 * Nx ? ix : ix - Mx, ky = iy < 2 * Ny ? iy : iy - My, kz = iz < 2 * Nz ? iz : iz - Mz;
        g[o] = make_double2(vg_GL(PI2 * kx / (Mx * hx), PI2 * ky / (My * hy), PI2 * kz / (Mz * hz), L), 0.0);
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

// In-place complex FFT of pencils: element i of pencil (i1, i2) at data[i1*s1 + i2*s2 + i*sa].
// grid.x = n1 * n2 pencils.
__global__ void k_fft_pencils(double2* __restrict__ data, int Lf, long sa, long n2, long s1, long s2,
                              int sign) {
    extern __shared__ double2 sm[];
    double2* a = sm;
    double2* b = sm + Lf;
    const long p = blockIdx.x;
    double2* base = data + (p / n2) * s1 + (p % n2) * s2;
    for (int i = threadIdx.x; i < Lf; i += blockDim.x) a[i] = base[(long)i * sa];
    double2* r = smem_fft_radix2(a, b, Lf, sign);
    for (int i = threadIdx.x; i < Lf; i += blockDim.x) base[(long)i * sa] = r[i];
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

// The same DCT-I for a TILE of C adjacent pencils per CTA (C even): pencils (a, b0 .. b0+C-1) of an
// nA x nB pencil grid; element k of pencil (a, b) at in[a*sA + b*sB + k*sK].  Two things make it several
// times faster than k_dct1_pencils: (1) two real-even pencils are packed as the real and imaginary part of
// ONE complex sequence -- both transforms are real, so they come out as Re and Im of the result; (2) the
// tile is chosen along the contiguous dimension, so that global accesses are full sectors; the twiddles
// come from a shared-memory table filled once per CTA.  Shared memory: [tw: Lf/2][a: C/2*Lf][b: C/2*Lf].
template <int C>
__global__ void k_dct1_tile(const double* __restrict__ in, double* __restrict__ out, int n, int nout,
                            long nB, long sA_in, long sB_in, long sK_in, long sA_out, long sB_out,
                            long sK_out, double scale) {
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
        const double v = c < nc ? src[(long)c * sB_in + (long)k * sK_in] : 0.0;
        const long sq = (long)(c >> 1) * Lf;
        af[2 * (sq + k) + (c & 1)] = v;
        if (k > 0 && k < n) af[2 * (sq + Lf - k) + (c & 1)] = v;
    }
    // Stockham autosort, all S sequences together: radix-4 stages (half the exchanges and barriers of radix 2),
    // then one radix-2 stage if log2(Lf) is odd.  Sign +: exp(+2 pi i ..); the input is real-even, so the sign
    // does not matter for the result.
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
    const double* rf = reinterpret_cast<const double*>(a);
    const int ototal = nout * C;
    for (int e = threadIdx.x; e < ototal; e += blockDim.x) {
        int d, c;
        if (sK_out == 1) { d = e % nout; c = e / nout; }
        else { c = e % C; d = e / C; }
        if (c < nc) dst[(long)c * sB_out + (long)d * sK_out] = scale * rf[2 * ((long)(c >> 1) * Lf + d) + (c & 1)];
    }
}

// VG: T[d] = scale * Re g[dx][dy][dz], d <= N, from the (4N)^3 complex grid
__global__ void k_restrict_vg(const double2* __restrict__ g, double* __restrict__ T, int Nx, int Ny,
                              int Nz, double scale) {
    const long total = (long)(Nx + 1) * (Ny + 1) * (Nz + 1);
    const long My = 4 * Ny, Mz = 4 * Nz;
    for (long o = blockIdx.x * (long)blockDim.x + threadIdx.x; o < total; o += (long)gridDim.x * blockDim.x) {
        const long dz = o % (Nz + 1), dy = (o / (Nz + 1)) % (Ny + 1), dx = o / ((long)(Nz + 1) * (Ny + 1));
        T[o] = scale * g[(dx * My + dy) * Mz + dz].x;
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

}  // namespace fsp

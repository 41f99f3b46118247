// fft_engine.cuh -- register-resident fp64 complex FFT for one "column" of M points spread over
// T = M/R threads (R points per thread), Stockham autosort, radix-{2,4,8,16} butterflies held in
// registers, one shared-memory exchange between stages.
//
// Index convention (validated against numpy in DESIGN.md "FFT engine"): thread t of a column holds
// v[i] <-> position t + T*i, both on entry (natural-order input) and on exit (natural-order
// output), so global loads/stores never need a transpose or a bit reversal.
//
// Stage with radix r after stages of total radix Ns (decimation in time):
//     butterfly j = t + T*m, m < R/r, works on v[m + i*(R/r)], i < r
//     k  = j mod Ns;  v[.] *= w_{Ns*r}^{i*k};  r-point DFT;
//     result i goes to position (j - k)*r + k + i*Ns.
//
// Forward sign is exp(-2 pi i ...).  The inverse transform is the same code with re/im swapped by
// the caller (IFFT(x) = swap(FFT(swap(x)))), so there is no second set of butterflies.
#pragma once
#include <cuda_runtime.h>

namespace fsp {

// ---- constants: w_32^k = cos(pi k/16) - i sin(pi k/16) (40-digit values, rounded by the compiler) ----
__device__ __forceinline__ double cos32(int k) {
    switch (k & 31) {
        case 0: return 1.0;
        case 1: case 31: return 0.980785280403230449126;
        case 2: case 30: return 0.923879532511286756128;
        case 3: case 29: return 0.831469612302545237079;
        case 4: case 28: return 0.707106781186547524401;
        case 5: case 27: return 0.555570233019602224743;
        case 6: case 26: return 0.382683432365089771728;
        case 7: case 25: return 0.195090322016128267848;
        case 8: case 24: return 0.0;
        case 9: case 23: return -0.195090322016128267848;
        case 10: case 22: return -0.382683432365089771728;
        case 11: case 21: return -0.555570233019602224743;
        case 12: case 20: return -0.707106781186547524401;
        case 13: case 19: return -0.831469612302545237079;
        case 14: case 18: return -0.923879532511286756128;
        case 15: case 17: return -0.980785280403230449126;
        default: return -1.0;
    }
}
__device__ __forceinline__ double sin32(int k) { return cos32(k - 8); }  // sin(x) = cos(x - pi/2)

// w_64^k = cos(pi k/32) - i sin(pi k/32) (the x tile kernels at Nx = 1024; even k reproduce cos32 bit for bit)
__device__ __forceinline__ double cos64(int k) {
    k &= 63;
    if (k > 32) k = 64 - k;            // cos is even
    const bool neg = k > 16;           // cos(pi - x) = -cos x
    if (neg) k = 32 - k;
    double v = 0.0;
    switch (k) {
        case 0: v = 1.0; break;
        case 1: v = 0.995184726672196886245; break;
        case 2: v = 0.980785280403230449126; break;
        case 3: v = 0.956940335732208864936; break;
        case 4: v = 0.923879532511286756128; break;
        case 5: v = 0.881921264348355029713; break;
        case 6: v = 0.831469612302545237079; break;
        case 7: v = 0.773010453362736960811; break;
        case 8: v = 0.707106781186547524401; break;
        case 9: v = 0.634393284163645498215; break;
        case 10: v = 0.555570233019602224743; break;
        case 11: v = 0.471396736825997648556; break;
        case 12: v = 0.382683432365089771728; break;
        case 13: v = 0.290284677254462367636; break;
        case 14: v = 0.195090322016128267848; break;
        case 15: v = 0.0980171403295606019942; break;
        default: v = 0.0; break;       // k = 16
    }
    return neg ? -v : v;
}
__device__ __forceinline__ double sin64(int k) { return cos64(k - 16); }

// ---- r-point DFT, in place, on elements re[0], re[S], re[2S], ... (natural order in and out) ---
template <int r, int S>
__device__ __forceinline__ void dft_pfa(double* re, double* im);

// r a power of two (decimation in time); dft_inplace below dispatches on r
template <int r, int S>
__device__ __forceinline__ void dft_pow2(double* re, double* im) {
    if constexpr (r == 2) {
        double ar = re[0], ai = im[0], br = re[S], bi = im[S];
        re[0] = ar + br; im[0] = ai + bi;
        re[S] = ar - br; im[S] = ai - bi;
    } else if constexpr (r > 2) {
        constexpr int H = r / 2;
        dft_pow2<H, 2 * S>(re, im);          // even-indexed inputs
        dft_pow2<H, 2 * S>(re + S, im + S);  // odd-indexed inputs
        double er[H], ei[H], qr[H], qi[H];
#pragma unroll
        for (int k = 0; k < H; ++k) {
            er[k] = re[2 * S * k]; ei[k] = im[2 * S * k];
            qr[k] = re[S + 2 * S * k]; qi[k] = im[S + 2 * S * k];
        }
#pragma unroll
        for (int k = 0; k < H; ++k) {
            if (k == 0) {
                re[0] = er[0] + qr[0]; im[0] = ei[0] + qi[0];
                re[S * H] = er[0] - qr[0]; im[S * H] = ei[0] - qi[0];
            } else if (4 * k == r) {  // w = -i:  q*w = qi - i qr
                re[S * k] = er[k] + qi[k]; im[S * k] = ei[k] - qr[k];
                re[S * (k + H)] = er[k] - qi[k]; im[S * (k + H)] = ei[k] + qr[k];
            } else {
                // w = c - i s.  q*w = c*[(qr + qi tn) + i (qi - qr tn)], tn = s/c     (|c| >= |s|)
                //                  = s*[(qr ct + qi) + i (qi ct - qr)], ct = c/s     (|c| <  |s|)
                // so twiddle + butterfly cost 6 FMAs instead of 8 (the constants fold at compile time).
                const double c = cos32(k * (32 / r)), s = sin32(k * (32 / r));
                double ur, ui, f;
                if (c * c >= s * s) {
                    const double tn = s / c;
                    ur = fma(qi[k], tn, qr[k]); ui = fma(-qr[k], tn, qi[k]); f = c;
                } else {
                    const double ct = c / s;
                    ur = fma(qr[k], ct, qi[k]); ui = fma(qi[k], ct, -qr[k]); f = s;
                }
                re[S * k] = fma(f, ur, er[k]); im[S * k] = fma(f, ui, ei[k]);
                re[S * (k + H)] = fma(-f, ur, er[k]); im[S * (k + H)] = fma(-f, ui, ei[k]);
            }
        }
    }
}

// ---- radices 3 and 5, and 6, 12, 10, 20 by the prime-factor algorithm (meshes 3 * 2^k, 5 * 2^k) ----
// Forward sign exp(-2 pi i ..).  Constants: sin(2 pi/3), cos/sin(2 pi/5), cos/sin(4 pi/5), 40 digits.
template <int S>
__device__ __forceinline__ void dft3(double* re, double* im) {
    constexpr double s3 = 0.8660254037844386467637231707529361834714;
    const double ar = re[S] + re[2 * S], ai = im[S] + im[2 * S], br = re[S] - re[2 * S], bi = im[S] - im[2 * S];
    const double tr = fma(-0.5, ar, re[0]), ti = fma(-0.5, ai, im[0]);
    re[0] += ar; im[0] += ai;
    // X1 = t - i s b,  X2 = t + i s b   (-i (br + i bi) = bi - i br)
    re[S] = fma(s3, bi, tr); im[S] = fma(-s3, br, ti);
    re[2 * S] = fma(-s3, bi, tr); im[2 * S] = fma(s3, br, ti);
}
template <int S>
__device__ __forceinline__ void dft5(double* re, double* im) {
    constexpr double c1 = 0.3090169943749474241022934171828190588602, c2 = -0.8090169943749474241022934171828190588602;
    constexpr double s1 = 0.9510565162951535721164393333793821434057, s2 = 0.5877852522924731291687059546390727685977;
    const double a1r = re[S] + re[4 * S], a1i = im[S] + im[4 * S], b1r = re[S] - re[4 * S], b1i = im[S] - im[4 * S];
    const double a2r = re[2 * S] + re[3 * S], a2i = im[2 * S] + im[3 * S], b2r = re[2 * S] - re[3 * S], b2i = im[2 * S] - im[3 * S];
    const double x0r = re[0], x0i = im[0];
    const double t1r = fma(c2, a2r, fma(c1, a1r, x0r)), t1i = fma(c2, a2i, fma(c1, a1i, x0i));
    const double t2r = fma(c1, a2r, fma(c2, a1r, x0r)), t2i = fma(c1, a2i, fma(c2, a1i, x0i));
    const double u1r = fma(s2, b2r, s1 * b1r), u1i = fma(s2, b2i, s1 * b1i);
    const double u2r = fma(-s1, b2r, s2 * b1r), u2i = fma(-s1, b2i, s2 * b1i);
    re[0] = x0r + a1r + a2r; im[0] = x0i + a1i + a2i;
    // X1 = t1 - i u1, X4 = t1 + i u1, X2 = t2 - i u2, X3 = t2 + i u2   (-i u = u.i - i u.r)
    re[S] = t1r + u1i; im[S] = t1i - u1r;
    re[4 * S] = t1r - u1i; im[4 * S] = t1i + u1r;
    re[2 * S] = t2r + u2i; im[2 * S] = t2i - u2r;
    re[3 * S] = t2r - u2i; im[3 * S] = t2i + u2r;
}

__host__ __device__ constexpr int mod_inverse(int a, int m) {   // a^-1 mod m (a, m coprime, m small)
    for (int x = 1; x < m; ++x)
        if ((a * x) % m == 1) return x;
    return 1;
}

// r = A * B with A in {2, 4}, B in {3, 5} coprime: Good-Thomas.  With n = (B n1 + A n2) mod r and k = k1 (mod A),
// k = k2 (mod B):  X[k] = sum_n1 w_A^(n1 k1) sum_n2 w_B^(n2 k2) x[n]  -- no twiddles between the two passes.
template <int r, int S>
__device__ __forceinline__ void dft_pfa(double* re, double* im) {
    constexpr int B = (r % 3 == 0) ? 3 : 5, A = r / B;
    static_assert(A * B == r && (A == 2 || A == 4), "prime-factor radices: 6, 12, 10, 20");
    double tr[r], ti[r];
    // pass 1: B-point transforms over n2 for each n1; result k2 kept in the slot (n1, k2)
#pragma unroll
    for (int n1 = 0; n1 < A; ++n1) {
        double ur[B], ui[B];
#pragma unroll
        for (int n2 = 0; n2 < B; ++n2) { ur[n2] = re[S * ((B * n1 + A * n2) % r)]; ui[n2] = im[S * ((B * n1 + A * n2) % r)]; }
        if constexpr (B == 3) dft3<1>(ur, ui); else dft5<1>(ur, ui);
#pragma unroll
        for (int k2 = 0; k2 < B; ++k2) { tr[n1 * B + k2] = ur[k2]; ti[n1 * B + k2] = ui[k2]; }
    }
    // pass 2: A-point transforms over n1 for each k2; X[k] with k = k1 (mod A), k = k2 (mod B) by the CRT
#pragma unroll
    for (int k2 = 0; k2 < B; ++k2) {
        double ur[A], ui[A];
#pragma unroll
        for (int n1 = 0; n1 < A; ++n1) { ur[n1] = tr[n1 * B + k2]; ui[n1] = ti[n1 * B + k2]; }
        dft_pow2<A, 1>(ur, ui);
#pragma unroll
        for (int k1 = 0; k1 < A; ++k1) {
            const int k = (k1 * B * mod_inverse(B % A, A) + k2 * A * mod_inverse(A % B, B)) % r;
            re[S * k] = ur[k1]; im[S * k] = ui[k1];
        }
    }
}

template <int r, int S>
__device__ __forceinline__ void dft_inplace(double* re, double* im) {
    if constexpr (r == 3) dft3<S>(re, im);
    else if constexpr (r == 5) dft5<S>(re, im);
    else if constexpr (r == 6 || r == 12 || r == 10 || r == 20) dft_pfa<r, S>(re, im);
    else dft_pow2<r, S>(re, im);
}

// ---- r-point DFT, strictly in place ------------------------------------------------------------
// Input x_i at re[S*i]; output X_k at re[S*brev_r(k)] (bit-reversed PLACEMENT, natural values): the
// iterative decimation-in-time network on the working array a[p] = element brev_r(p), whose butterflies
// (a[q], a[q+h]) -> (a[q] + w a[q+h], a[q] - w a[q+h]) overwrite their own operands, so the live set is
// the 2r data registers plus two temporaries per butterfly in flight (the recursive dft_inplace above
// gathers copies at every level and needs half as many registers again).  All indices are compile-time.
__host__ __device__ constexpr int brev(int v, int r) {
    int o = 0;
    for (int b = 1; b < r; b <<= 1) { o = (o << 1) | (v & 1); v >>= 1; }
    return o;
}

// LO..HI: the radix-2 levels (butterfly spans len = LO, 2 LO, .., HI) that are executed; the full transform is
// LO = 2, HI = r.  Splitting off the first level lets a caller prune it (fft2_padded_pass).
template <int r, int S, int LO = 2, int HI = r>
__device__ __forceinline__ void dft_br(double* re, double* im) {
#pragma unroll
    for (int len = LO; len <= HI; len *= 2) {
        const int half = len / 2;
#pragma unroll
        for (int blk = 0; blk < r; blk += len) {
#pragma unroll
            for (int k = 0; k < half; ++k) {
                const int p = S * brev(blk + k, r), q = S * brev(blk + k + half, r);
                const double ar = re[p], ai = im[p], br = re[q], bi = im[q];
                if (k == 0) {
                    re[p] = ar + br; im[p] = ai + bi; re[q] = ar - br; im[q] = ai - bi;
                } else if (4 * k == len) {  // w = -i
                    re[p] = ar + bi; im[p] = ai - br; re[q] = ar - bi; im[q] = ai + br;
                } else {
                    const double c = cos32(k * (32 / len)), s = sin32(k * (32 / len));
                    double ur, ui, f;
                    if (c * c >= s * s) {
                        const double tn = s / c;
                        ur = fma(bi, tn, br); ui = fma(-br, tn, bi); f = c;
                    } else {
                        const double ct = c / s;
                        ur = fma(br, ct, bi); ui = fma(bi, ct, -br); f = s;
                    }
                    re[q] = fma(-f, ur, ar); im[q] = fma(-f, ui, ai);
                    re[p] = fma(f, ur, ar); im[p] = fma(f, ui, ai);
                }
            }
        }
    }
}

// ---- static description of one FFT size ---------------------------------------------------------
// R points per thread; up to three stages r1*r2*r3 = M (r = 1 marks "no stage").
template <int M_, int R_, int R1_, int R2_, int R3_>
struct FftCfgT {
    static constexpr int M = M_, R = R_, R1 = R1_, R2 = R2_, R3 = R3_, T = M_ / R_;
    static_assert(R1_ * R2_ * R3_ == M_, "radices must multiply to M");
    static_assert(R_ % R1_ == 0 && R_ % R2_ == 0 && R_ % R3_ == 0, "radix must divide R");
};
template <int M> struct FftCfg;
template <> struct FftCfg<4> : FftCfgT<4, 4, 4, 1, 1> {};
template <> struct FftCfg<8> : FftCfgT<8, 8, 8, 1, 1> {};
template <> struct FftCfg<16> : FftCfgT<16, 16, 16, 1, 1> {};
template <> struct FftCfg<32> : FftCfgT<32, 8, 8, 4, 1> {};
template <> struct FftCfg<64> : FftCfgT<64, 8, 8, 8, 1> {};
template <> struct FftCfg<128> : FftCfgT<128, 16, 16, 8, 1> {};
template <> struct FftCfg<256> : FftCfgT<256, 16, 16, 16, 1> {};
template <> struct FftCfg<512> : FftCfgT<512, 8, 8, 8, 8> {};
template <> struct FftCfg<1024> : FftCfgT<1024, 16, 16, 16, 4> {};
// 3 * 2^k and 5 * 2^k: power-of-two stages first (the scatter of a stage assumes that the radices
// before it multiply to a power of two), the stage that carries the factor 3 or 5 last
template <> struct FftCfg<6> : FftCfgT<6, 6, 6, 1, 1> {};
template <> struct FftCfg<12> : FftCfgT<12, 12, 12, 1, 1> {};
template <> struct FftCfg<24> : FftCfgT<24, 12, 2, 12, 1> {};
template <> struct FftCfg<48> : FftCfgT<48, 12, 4, 12, 1> {};
template <> struct FftCfg<96> : FftCfgT<96, 12, 4, 2, 12> {};
template <> struct FftCfg<192> : FftCfgT<192, 12, 4, 4, 12> {};
template <> struct FftCfg<384> : FftCfgT<384, 24, 8, 4, 12> {};
template <> struct FftCfg<768> : FftCfgT<768, 24, 8, 8, 12> {};
template <> struct FftCfg<10> : FftCfgT<10, 10, 10, 1, 1> {};
template <> struct FftCfg<20> : FftCfgT<20, 20, 20, 1, 1> {};
template <> struct FftCfg<40> : FftCfgT<40, 20, 2, 20, 1> {};
template <> struct FftCfg<80> : FftCfgT<80, 20, 4, 20, 1> {};
template <> struct FftCfg<160> : FftCfgT<160, 20, 4, 2, 20> {};
template <> struct FftCfg<320> : FftCfgT<320, 20, 4, 4, 20> {};

// ---- one stage: twiddle (if Ns > 1) and butterflies ----------------------------------------------
// W: table of exp(-2 pi i n / LTAB), n < LTAB, in shared memory; LTAB a multiple of Ns*r.
template <int M, int R, int r, int Ns, int LTAB>
__device__ __forceinline__ void fft_stage(double (&re)[R], double (&im)[R], int t,
                                          const double2* __restrict__ W) {
    constexpr int T = M / R, nb = R / r;
#pragma unroll
    for (int m = 0; m < nb; ++m) {
        if constexpr (Ns > 1) {
            const int k = (t + T * m) & (Ns - 1);
            constexpr int step = LTAB / (Ns * r);
#pragma unroll
            for (int i = 1; i < r; ++i) {
                const double2 w = W[i * k * step];
                const double xr = re[m + i * nb], xi = im[m + i * nb];
                re[m + i * nb] = xr * w.x - xi * w.y;
                im[m + i * nb] = xr * w.y + xi * w.x;
            }
        }
        dft_inplace<r, nb>(&re[m], &im[m]);
    }
}

// scatter the results of a stage to their Stockham positions in the exchange buffer
// buf: this column's buffer; element at position p lives at buf[p * PS].
template <int M, int R, int r, int Ns, int PS>
__device__ __forceinline__ void fft_exchange_write(const double (&re)[R], const double (&im)[R], int t,
                                                   double2* __restrict__ buf) {
    constexpr int T = M / R, nb = R / r;
#pragma unroll
    for (int m = 0; m < nb; ++m) {
        const int j = t + T * m;
        const int k = j & (Ns - 1);
        const int j0 = (j - k) * r + k;
#pragma unroll
        for (int i = 0; i < r; ++i) buf[(j0 + i * Ns) * PS] = make_double2(re[m + i * nb], im[m + i * nb]);
    }
}

template <int M, int R, int PS>
__device__ __forceinline__ void fft_exchange_read(double (&re)[R], double (&im)[R], int t,
                                                  const double2* __restrict__ buf) {
    constexpr int T = M / R;
#pragma unroll
    for (int i = 0; i < R; ++i) {
        const double2 v = buf[(t + T * i) * PS];
        re[i] = v.x; im[i] = v.y;
    }
}

// ---- the whole M-point forward FFT of one column --------------------------------------------------
// All threads of the CTA must call this together (it contains __syncthreads()).
// On return the exchange buffer may be reused immediately by the caller only after a barrier;
// the function itself places a barrier before each of its own writes.
template <class Cfg, int PS, int LTAB>
__device__ __forceinline__ void fft_forward(double (&re)[Cfg::R], double (&im)[Cfg::R], int t,
                                            double2* __restrict__ buf, const double2* __restrict__ W) {
    constexpr int M = Cfg::M, R = Cfg::R;
    fft_stage<M, R, Cfg::R1, 1, LTAB>(re, im, t, W);
    if constexpr (Cfg::R2 > 1) {
        __syncthreads();  // previous readers of buf are done
        fft_exchange_write<M, R, Cfg::R1, 1, PS>(re, im, t, buf);
        __syncthreads();
        fft_exchange_read<M, R, PS>(re, im, t, buf);
        fft_stage<M, R, Cfg::R2, Cfg::R1, LTAB>(re, im, t, W);
    }
    if constexpr (Cfg::R3 > 1) {
        __syncthreads();
        fft_exchange_write<M, R, Cfg::R2, Cfg::R1, PS>(re, im, t, buf);
        __syncthreads();
        fft_exchange_read<M, R, PS>(re, im, t, buf);
        fft_stage<M, R, Cfg::R3, Cfg::R1 * Cfg::R2, LTAB>(re, im, t, W);
    }
}

// unnormalised inverse: swap the roles of re and im
template <class Cfg, int PS, int LTAB>
__device__ __forceinline__ void fft_inverse(double (&re)[Cfg::R], double (&im)[Cfg::R], int t,
                                            double2* __restrict__ buf, const double2* __restrict__ W) {
    // the exchange then stores (im, re) pairs -- harmless, it is read back the same way
    fft_forward<Cfg, PS, LTAB>(im, re, t, buf, W);
}

}  // namespace fsp

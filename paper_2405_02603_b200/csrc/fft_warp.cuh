// fft_warp.cuh -- two-stage, single-exchange fp64 complex FFT of M = R1*R2 points held by a group of
// T = M/R lanes of ONE warp (R = max(R1, R2) points per lane).  Built for the three roofs a B200 SM
// puts on an fp64 FFT at once: 64 fp64 ops/clk, 128 B/clk of shared
// memory, and its share of HBM.  Compared with the three-stage engine of fft_engine.cuh:
//   * one shared-memory exchange per transform instead of two (half the shared-memory bytes),
//   * the exchange is private to the lane group, so only __syncwarp() is needed, never a CTA barrier,
//   * the exchange buffer is padded by one element per R1 so that both the strided writes and the
//     unit-stride reads are bank-conflict free for 16-byte accesses (8 lanes = 128 B per wavefront),
//   * the stage-2 twiddles come from a 2-D table tw[i][j] = w_M^(i*j) that lanes read at unit stride.
//
// Index convention (same as fft_engine.cuh): lane t holds v[i] <-> position t + T*i, natural order on
// entry and on exit.
//   stage 1: nb1 = R/R1 butterflies per lane; butterfly j = t + T*m works on v[m + i*nb1], i < R1
//            (positions j + (M/R1)*i), no twiddles; result i goes to position j*R1 + i.
//   stage 2: nb2 = R/R2 butterflies per lane; butterfly j = t + T*m (j < R1) works on v[m + i*nb2],
//            i < R2 (positions j + R1*i), input i multiplied by w_M^(i*j) first; result i is the
//            output at position j + R1*i = t + T*(m + i*nb2): the register it already sits in.
#pragma once
#include "fft_engine.cuh"

namespace fsp {

template <int M_, int R1_, int R2_>
struct Fft2CfgT {
    static constexpr int M = M_, R1 = R1_, R2 = R2_;
    static constexpr int R = R1_ > R2_ ? R1_ : R2_;
    static constexpr int T = M_ / R;
    static constexpr int NB1 = R / R1_, NB2 = R / R2_;
    static constexpr int BUF = M_ + M_ / R1_;  // padded exchange buffer, in double2 elements
    static_assert(R1_ * R2_ == M_, "radices must multiply to M");
    static_assert(T >= 1 && T <= 16, "a lane group must fit half a warp");
};
template <int M> struct Fft2Cfg;
template <> struct Fft2Cfg<8> : Fft2CfgT<8, 4, 2> {};
template <> struct Fft2Cfg<16> : Fft2CfgT<16, 4, 4> {};
template <> struct Fft2Cfg<32> : Fft2CfgT<32, 8, 4> {};
template <> struct Fft2Cfg<64> : Fft2CfgT<64, 8, 8> {};
template <> struct Fft2Cfg<128> : Fft2CfgT<128, 16, 8> {};
template <> struct Fft2Cfg<256> : Fft2CfgT<256, 16, 16> {};
template <> struct Fft2Cfg<512> : Fft2CfgT<512, 16, 32> {};

// padded address of position p (one pad element after every R1 positions)
template <int R1>
__device__ __forceinline__ int pad_pos(int p) { return p + p / R1; }

// Forward transform (sign exp(-2 pi i ..)).  buf: this lane group's exchange buffer (Cfg::BUF double2);
// tw: table tw[i*R1 + j] = exp(-2 pi i * i*j / M), i < R2, j < R1 (shared memory).
// All 32 lanes of the warp must call this together.
template <class Cfg>
__device__ __forceinline__ void fft2_forward(double (&re)[Cfg::R], double (&im)[Cfg::R], int t,
                                             double2* __restrict__ buf, const double2* __restrict__ tw) {
    constexpr int R = Cfg::R, R1 = Cfg::R1, R2 = Cfg::R2, T = Cfg::T, NB1 = Cfg::NB1, NB2 = Cfg::NB2;
#pragma unroll
    for (int m = 0; m < NB1; ++m) dft_inplace<R1, NB1>(&re[m], &im[m]);
    __syncwarp();  // earlier readers of buf are done
#pragma unroll
    for (int m = 0; m < NB1; ++m) {
        double2* dst = buf + (t + T * m) * (R1 + 1);
#pragma unroll
        for (int i = 0; i < R1; ++i) dst[i] = make_double2(re[m + i * NB1], im[m + i * NB1]);
    }
    __syncwarp();
#pragma unroll
    for (int i = 0; i < R; ++i) {
        // position p = t + T*i; p / R1 is a compile-time constant when T divides R1 (t < T <= R1)
        int a;
        if constexpr (R1 % T == 0) a = t + T * i + (T * i) / R1;
        else a = pad_pos<R1>(t + T * i);
        const double2 v = buf[a];
        re[i] = v.x; im[i] = v.y;
    }
#pragma unroll
    for (int m = 0; m < NB2; ++m) {
#pragma unroll
        for (int i = 1; i < R2; ++i) {
            const double2 w = tw[i * R1 + t + T * m];
            const double xr = re[m + i * NB2], xi = im[m + i * NB2];
            re[m + i * NB2] = xr * w.x - xi * w.y;
            im[m + i * NB2] = xr * w.y + xi * w.x;
        }
        dft_inplace<R2, NB2>(&re[m], &im[m]);
    }
}

// unnormalised inverse: swap the roles of re and im (IFFT(x) = swap(FFT(swap(x))))
template <class Cfg>
__device__ __forceinline__ void fft2_inverse(double (&re)[Cfg::R], double (&im)[Cfg::R], int t,
                                             double2* __restrict__ buf, const double2* __restrict__ tw) {
    fft2_forward<Cfg>(im, re, t, buf, tw);
}

}  // namespace fsp

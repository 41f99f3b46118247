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
#include "tma.cuh"

namespace fsp {

template <int M_, int R1_, int R2_>
struct Fft2CfgT {
    static constexpr int M = M_, R1 = R1_, R2 = R2_;
    static constexpr int R = R1_ > R2_ ? R1_ : R2_;
    static constexpr int T = M_ / R;
    static constexpr int NB1 = R / R1_, NB2 = R / R2_;
    static constexpr int BUF = M_ + M_ / R1_;  // padded exchange buffer, in double2 elements
    static_assert(R1_ * R2_ == M_, "radices must multiply to M");
    static_assert(T >= 1 && T <= 32, "a lane group must fit a warp");
};
template <int M> struct Fft2Cfg;
template <> struct Fft2Cfg<8> : Fft2CfgT<8, 4, 2> {};
template <> struct Fft2Cfg<16> : Fft2CfgT<16, 4, 4> {};
template <> struct Fft2Cfg<32> : Fft2CfgT<32, 8, 4> {};
template <> struct Fft2Cfg<64> : Fft2CfgT<64, 8, 8> {};
template <> struct Fft2Cfg<128> : Fft2CfgT<128, 16, 8> {};
template <> struct Fft2Cfg<256> : Fft2CfgT<256, 16, 16> {};
template <> struct Fft2Cfg<512> : Fft2CfgT<512, 16, 32> {};
template <> struct Fft2Cfg<1024> : Fft2CfgT<1024, 32, 32> {};   // one branch per warp (k_conv_z_p)

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

// ---- stage 2 with lane-constant twiddles ------------------------------------------------------------
// The stage-2 butterfly j computes  Y_k = sum_i x_i om^i w_R2^(i k),  om = w_M^j  (the input twiddles of
// fft2_forward folded into the transform: a DFT at the shifted frequencies k + j/R1).  Decimation in time
// keeps that form at every level: with b_r = om^(R2/r),
//     Y_k = E_k + (b_r w_r^k) O_k,   Y_(k+r/2) = E_k - (b_r w_r^k) O_k,   k < r/2,
// E, O the size-r/2 transforms (base b_r^2) of the even / odd inputs.  Since w_r^(k + r/4) = -i w_r^k, a
// size-r level needs only max(1, r/4) distinct twiddles b_r w_r^k, R2/2 in total over all levels.  They
// depend on j only, i.e. they are per-lane constants for the whole kernel: held in registers as
// (cos, tan) pairs, each twiddle + butterfly is 6 FMAs and stage 2 reads no twiddle table at all
// (the LSU data pipe, not HBM, is the first roof of these kernels).
// Constant i of level r (r >= 4) sits at index r/4 + (k mod r/4); level 2 at index 0.
template <int R2> struct LaneTw { static constexpr int NC = R2 >= 4 ? R2 / 2 : 1; };

template <int r, int S>
__device__ __forceinline__ void dft_lane(double* re, double* im, const double* __restrict__ cc,
                                         const double* __restrict__ tn) {
    // in place: input x_i at re[S*brev_r(i)] (the caller loads it there), output Y_k at re[S*k].
    // Butterflies are emitted in batches of BT: first the 2*BT twiddle products, then the 4*BT sums, so
    // that no FMA directly follows the one it depends on (one warp alone must keep the fp64 pipe fed).
    constexpr int BT = (r / 2 < 4) ? r / 2 : 4;
#pragma unroll
    for (int len = 2; len <= r; len *= 2) {
        const int half = len / 2;
        const int OFS = len >= 4 ? len / 4 : 0, Q = len >= 4 ? len / 4 : 1;
#pragma unroll
        for (int b0 = 0; b0 < r / 2; b0 += BT) {
            double ur[BT], ui[BT];
#pragma unroll
            for (int j = 0; j < BT; ++j) {
                const int bb = b0 + j, k = bb % half, blk = (bb / half) * len;
                const int q = S * (blk + k + half);
                const double tg = tn[OFS + (k % Q)];
                // b (c - i s) = c [(br + bi tg) + i (bi - br tg)],  tg = s / c
                ur[j] = fma(im[q], tg, re[q]);
                ui[j] = fma(-re[q], tg, im[q]);
            }
#pragma unroll
            for (int j = 0; j < BT; ++j) {
                const int bb = b0 + j, k = bb % half, blk = (bb / half) * len;
                const int p = S * (blk + k), q = S * (blk + k + half);
                const double c = cc[OFS + (k % Q)];
                const double ar = re[p], ai = im[p];
                if (((k / Q) & 1) == 0) {
                    re[q] = fma(-c, ur[j], ar); im[q] = fma(-c, ui[j], ai);
                    re[p] = fma(c, ur[j], ar); im[p] = fma(c, ui[j], ai);
                } else {  // twiddle times -i:  c (ui - i ur)
                    re[q] = fma(-c, ui[j], ar); im[q] = fma(c, ur[j], ai);
                    re[p] = fma(c, ui[j], ar); im[p] = fma(-c, ur[j], ai);
                }
            }
        }
    }
}

// fft2_forward with the lane-constant stage 2 and in-place butterflies.
// Natural order in and out (lane t holds position t + T*i in register i): stage 1 leaves output k of
// butterfly m in register m + NB1*brev(k), which is where the exchange write takes it from; the exchange
// read puts input e of stage-2 butterfly m into register m + NB2*brev(e), so that the in-place stage 2
// ends in natural order.  cc/tn: [NB2][LaneTw<R2>::NC] constants of this lane's butterflies j = t + T*m
// (host table make_lane_table, loaded once per kernel).
template <class Cfg>
__device__ __forceinline__ void fft2_forward_lc(double (&re)[Cfg::R], double (&im)[Cfg::R], int t,
                                                double2* __restrict__ buf,
                                                const double (&cc)[Cfg::NB2][LaneTw<Cfg::R2>::NC],
                                                const double (&tn)[Cfg::NB2][LaneTw<Cfg::R2>::NC]) {
    constexpr int R = Cfg::R, R1 = Cfg::R1, R2 = Cfg::R2, T = Cfg::T, NB1 = Cfg::NB1, NB2 = Cfg::NB2;
    __syncwarp();  // earlier readers of buf are done (placed first so that the stores of one stage-1
                   // butterfly can drain while the next one is computed)
#pragma unroll
    for (int m = 0; m < NB1; ++m) {
        dft_br<R1, NB1>(&re[m], &im[m]);
        double2* dst = buf + (t + T * m) * (R1 + 1);
#pragma unroll
        for (int i = 0; i < R1; ++i)   // output i of butterfly m sits in register m + NB1*brev(i)
            dst[i] = make_double2(re[m + brev(i, R1) * NB1], im[m + brev(i, R1) * NB1]);
    }
    __syncwarp();
#pragma unroll
    for (int i = 0; i < R; ++i) {
        int a;
        if constexpr (R1 % T == 0) a = t + T * i + (T * i) / R1;
        else a = pad_pos<R1>(t + T * i);
        const double2 v = buf[a];
        const int d = (i % NB2) + NB2 * brev(i / NB2, R2);
        re[d] = v.x; im[d] = v.y;
    }
#pragma unroll
    for (int m = 0; m < NB2; ++m) dft_lane<R2, NB2>(&re[m], &im[m], cc[m], tn[m]);
}

// The same transform for the tile kernels (strided axes): a GROUP of CW*T threads transforms CW adjacent
// columns at once, thread (c, t) = (column, lane of the column), c fastest, so that a quarter-warp is
// 8 columns of one position: every exchange access is one contiguous 128-byte row of the buffer
// E[position][CW] (conflict free without padding) and every global access a full line.  The T lanes of
// a column sit in different warps, so the two syncs are named barriers over the group.
// Ec = E + c;  bar_id: the group's barrier.
template <class Cfg, int CW>
__device__ __forceinline__ void fft2_forward_tile(double (&re)[Cfg::R], double (&im)[Cfg::R], int t,
                                                  double2* __restrict__ Ec, int bar_id,
                                                  const double (&cc)[Cfg::NB2][LaneTw<Cfg::R2>::NC],
                                                  const double (&tn)[Cfg::NB2][LaneTw<Cfg::R2>::NC]) {
    constexpr int R = Cfg::R, R1 = Cfg::R1, R2 = Cfg::R2, T = Cfg::T, NB1 = Cfg::NB1, NB2 = Cfg::NB2;
#pragma unroll
    for (int m = 0; m < NB1; ++m) dft_br<R1, NB1>(&re[m], &im[m]);
    bar_sync(bar_id, CW * T);  // earlier readers of E are done
#pragma unroll
    for (int m = 0; m < NB1; ++m) {
        double2* dst = Ec + (t + T * m) * (R1 * CW);
#pragma unroll
        for (int i = 0; i < R1; ++i)
            dst[i * CW] = make_double2(re[m + brev(i, R1) * NB1], im[m + brev(i, R1) * NB1]);
    }
    bar_sync(bar_id, CW * T);
#pragma unroll
    for (int i = 0; i < R; ++i) {
        const double2 v = Ec[(t + T * i) * CW];
        const int d = (i % NB2) + NB2 * brev(i / NB2, R2);
        re[d] = v.x; im[d] = v.y;
    }
#pragma unroll
    for (int m = 0; m < NB2; ++m) dft_lane<R2, NB2>(&re[m], &im[m], cc[m], tn[m]);
}

// unnormalised inverse: swap the roles of re and im (IFFT(x) = swap(FFT(swap(x))))
template <class Cfg>
__device__ __forceinline__ void fft2_inverse(double (&re)[Cfg::R], double (&im)[Cfg::R], int t,
                                             double2* __restrict__ buf, const double2* __restrict__ tw) {
    fft2_forward<Cfg>(im, re, t, buf, tw);
}

}  // namespace fsp

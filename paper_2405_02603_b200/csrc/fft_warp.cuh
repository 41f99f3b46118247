// fft_warp.cuh -- two-stage, single-exchange fp64 complex FFT of M = R1*R2 points held by a group of
// T = M/R lanes of ONE warp (R = max(R1, R2) points per lane).  Built for the three roofs a B200 SM
// puts on an fp64 FFT at once: 64 fp64 ops/clk, 128 B/clk of shared
// memory, and its share of HBM.  Compared with the three-stage engine of fft_engine.cuh:
//   * one shared-memory exchange per transform instead of two (half the shared-memory bytes),
//   * the exchange is private to the lane group, so only __syncwarp() is needed, never a CTA barrier,
//   * the exchange buffer is padded by one element per R1 so that both the strided writes and the
//     unit-stride reads are bank-conflict free for 16-byte accesses (8 lanes = 128 B per wavefront),
//   * the stage-2 twiddles are lane constants held in registers (dft_lane below): no table is read.
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

// ---- stage 2 with lane-constant twiddles ------------------------------------------------------------
// The stage-2 butterfly j computes  Y_k = sum_i x_i om^i w_R2^(i k),  om = w_M^j  (the input twiddles of
// two-stage scheme folded into the transform: a DFT at the shifted frequencies k + j/R1).  Decimation in time
// keeps that form at every level: with b_r = om^(R2/r),
//     Y_k = E_k + (b_r w_r^k) O_k,   Y_(k+r/2) = E_k - (b_r w_r^k) O_k,   k < r/2,
// E, O the size-r/2 transforms (base b_r^2) of the even / odd inputs.  Since w_r^(k + r/4) = -i w_r^k, a
// size-r level needs only max(1, r/4) distinct twiddles b_r w_r^k, R2/2 in total over all levels.  They
// depend on j only, i.e. they are per-lane constants for the whole kernel: held in registers as
// (cos, tan) pairs, each twiddle + butterfly is 6 FMAs and stage 2 reads no twiddle table at all
// (the LSU data pipe, not HBM, is the first roof of these kernels).
// Constant i of level r (r >= 4) sits at index r/4 + (k mod r/4); level 2 at index 0.
template <int R2> struct LaneTw { static constexpr int NC = R2 >= 4 ? R2 / 2 : 1; };

// LO..HI: the levels executed (full transform: 2..r).  HALF_OUT (only meaningful when HI == r): only the outputs
// Y_k, k < r/2, of the last level are formed (4 instead of 6 fp64 instructions per butterfly): the output-pruned
// inverse of a padded pencil, whose second half is discarded.
template <int r, int S, int LO = 2, int HI = r, bool HALF_OUT = false>
__device__ __forceinline__ void dft_lane(double* re, double* im, const double* __restrict__ cc,
                                         const double* __restrict__ tn) {
    // in place: input x_i at re[S*brev_r(i)] (the caller loads it there), output Y_k at re[S*k].
    // Butterflies are emitted in batches of BT: first the 2*BT twiddle products, then the 4*BT sums, so
    // that no FMA directly follows the one it depends on (one warp alone must keep the fp64 pipe fed).
    constexpr int BT = (r / 2 < 4) ? r / 2 : 4;
#pragma unroll
    for (int len = LO; len <= HI; len *= 2) {
        const int half = len / 2;
        const int OFS = len >= 4 ? len / 4 : 0, Q = len >= 4 ? len / 4 : 1;
        const bool only_p = HALF_OUT && len == r;
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
                    if (!only_p) { re[q] = fma(-c, ur[j], ar); im[q] = fma(-c, ui[j], ai); }
                    re[p] = fma(c, ur[j], ar); im[p] = fma(c, ui[j], ai);
                } else {  // twiddle times -i:  c (ui - i ur)
                    if (!only_p) { re[q] = fma(-c, ui[j], ar); im[q] = fma(c, ur[j], ai); }
                    re[p] = fma(c, ui[j], ar); im[p] = fma(-c, ur[j], ai);
                }
            }
        }
    }
}

// The two-stage transform with the lane-constant stage 2 and in-place butterflies.
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

// ---- the two passes of a zero-padded pencil of Cfg::M = 2 Nz points in ONE lane group (k_conv_z_f) ------------
// pass 0 (forward, input-pruned): the inputs at positions >= M/2 (registers i >= R/2) are zero, so the first
//   radix-2 level of stage 1, (x_i, 0) -> (x_i, x_i), is a register copy (the zero half of rho2 is
//   never read): the CALLER loads x_i into registers i and i + R/2 and the level is skipped;
// pass 1 (inverse by IFFT(Y) = conj(FFT(conj Y)), output-pruned): only the outputs at positions < M/2 (registers
//   k < R/2) are kept, so the last level of stage 2 forms only those.
// Everything between is ONE copy of the code for both passes (two unrolled copies overflow the instruction cache).
// Compared with two half-length branches per pencil (k_conv_z_p): the same exchange volume, but no pre-twiddle,
// no final combine, no hand-over between warps and one global read of the pencil instead of two: 30 % fewer
// shared-memory / L1 wavefronts, which is the first roof of this pass.
template <class Cfg>
__device__ __forceinline__ void fft2_padded_pass(double (&re)[Cfg::R], double (&im)[Cfg::R], int t,
                                                 double2* __restrict__ buf,
                                                 const double (&cc)[LaneTw<Cfg::R2>::NC],
                                                 const double (&tn)[LaneTw<Cfg::R2>::NC], int pass) {
    constexpr int R = Cfg::R, R1 = Cfg::R1, R2 = Cfg::R2, T = Cfg::T, NB1 = Cfg::NB1, NB2 = Cfg::NB2;
    static_assert(NB2 == 1, "the output pruning assumes one stage-2 butterfly per lane");
    __syncwarp();  // earlier readers of buf are done
    if (pass != 0) {   // pass 0: the caller has already put x_i into the register of x_(i + R1/2) = 0 (see above)
#pragma unroll
        for (int m = 0; m < NB1; ++m) dft_br<R1, NB1, 2, 2>(&re[m], &im[m]);
    }
#pragma unroll
    for (int m = 0; m < NB1; ++m) {
        dft_br<R1, NB1, 4, R1>(&re[m], &im[m]);
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
        const int d = brev(i, R2);
        re[d] = v.x; im[d] = v.y;
    }
    dft_lane<R2, 1, 2, R2 / 2>(re, im, cc, tn);
    if (pass == 0) dft_lane<R2, 1, R2, R2, false>(re, im, cc, tn);
    else dft_lane<R2, 1, R2, R2, true>(re, im, cc, tn);
}

// ---- 512 points over ALL 32 lanes of a warp, 16 points per lane (k_conv_z_s) ---------------------------
// 512 = 32 x 16 with the radix-32 stage split over lane pairs (l, l ^ 16): lane l = j + 16 h holds the inputs
// x[j + 16 i], i = 2 i' + h, of stage-1 butterfly j (positions l + 32 i': the natural layout, T = 32), runs the
// radix-16 sub-transform of its own 16 inputs in registers (E_k on h = 0, O_k on h = 1) and the last radix-2 level
//     Y_k = E_k + w_32^k O_k,   Y_(k+16) = E_k - w_32^k O_k
// is shared by the pair through warp shuffles: lane h finishes k = m + 8 h, m < 8, so each lane sends 8 values and
// receives 8 (32 SHFL.32) instead of a second trip through shared memory.  Stage 2 is one radix-16 butterfly per
// lane with lane-constant twiddles (dft_lane).  Half the registers of Fft2Cfg<512> (16 x 32 over 16 lanes, 32
// points per lane): 16 warps per SM instead of 8 keep the fp64 pipe and the shared-memory pipe busy at the same
// time.  Natural order in and out: register i <-> position lane + 32 i.
struct Fft512S {
    static constexpr int M = 512, R = 16, T = 32, R1 = 32, R2 = 16, NB2 = 1;
    static constexpr int BUF = M + M / R1;   // one pad element per R1 positions
    static constexpr int NC = LaneTw<R2>::NC;
    static constexpr int NX = 8;             // lane constants of the shuffled level: w_32^(m + 8 h), m < 8
};

// xc/xt: (cos, tan) of w_32^(m + 8 h) for this lane's h = lane >> 4
__device__ __forceinline__ void fft512s_forward(double (&re)[16], double (&im)[16], int lane, double2* __restrict__ buf,
                                                const double (&cc)[Fft512S::NC], const double (&tn)[Fft512S::NC],
                                                const double (&xc)[8], const double (&xt)[8]) {
    const bool h = lane >= 16;
    __syncwarp();   // earlier readers of buf are done
    dft_br<16, 1>(re, im);   // output k of the sub-transform sits in register brev(k, 16)
    double2* dst = buf + (lane & 15) * 33 + (h ? 8 : 0);   // stage-1 output k of butterfly j -> padded position 33 j + k
#pragma unroll
    for (int m = 0; m < 8; ++m) {
        const int r0 = brev(m, 16), r1 = brev(m + 8, 16);
        // h = 0 keeps E_m (r0) and gives E_(m+8) (r1); h = 1 keeps O_(m+8) (r1) and gives O_m (r0)
        const double sr = h ? re[r0] : re[r1], si = h ? im[r0] : im[r1];
        const double kr = h ? re[r1] : re[r0], ki = h ? im[r1] : im[r0];
        const double pr = __shfl_xor_sync(0xffffffffu, sr, 16), pi = __shfl_xor_sync(0xffffffffu, si, 16);
        const double ar = h ? pr : kr, ai = h ? pi : ki;   // E_(m + 8 h)
        const double br = h ? kr : pr, bi = h ? ki : pi;   // O_(m + 8 h)
        const double ur = fma(bi, xt[m], br), ui = fma(-br, xt[m], bi);
        const double y0r = fma(xc[m], ur, ar), y0i = fma(xc[m], ui, ai);      // Y_(m + 8 h)
        const double y1r = fma(-xc[m], ur, ar), y1i = fma(-xc[m], ui, ai);    // Y_(m + 8 h + 16)
        dst[m] = make_double2(y0r, y0i);
        dst[m + 16] = make_double2(y1r, y1i);
    }
    __syncwarp();
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const double2 v = buf[lane + 33 * i];   // position lane + 32 i
        re[brev(i, 16)] = v.x; im[brev(i, 16)] = v.y;
    }
    dft_lane<16, 1>(re, im, cc, tn);
}

// The same transform for the tile kernels (strided axes): a GROUP of CW*T threads transforms CW adjacent
// columns at once, thread (c, t) = (column, lane of the column), c fastest, so that a quarter-warp is
// 8 columns of one position: every exchange access is one contiguous 128-byte row of the buffer
// E[position][CW] (conflict free without padding) and every global access a full line.  The T lanes of
// a column sit in different warps, so the two syncs are named barriers over the group.
// Ec = E + c;  bar_id: the group's barrier.
// LO1 = 4: the first radix-2 level of stage 1 is skipped (zero-padded input: the caller has put x_i into the register
// of x_(i + R1/2) = 0, see fft2_padded_pass).
template <class Cfg, int CW, int LO1 = 2>
__device__ __forceinline__ void fft2_forward_tile(double (&re)[Cfg::R], double (&im)[Cfg::R], int t,
                                                  double2* __restrict__ Ec, int bar_id,
                                                  const double (&cc)[Cfg::NB2][LaneTw<Cfg::R2>::NC],
                                                  const double (&tn)[Cfg::NB2][LaneTw<Cfg::R2>::NC]) {
    constexpr int R = Cfg::R, R1 = Cfg::R1, R2 = Cfg::R2, T = Cfg::T, NB1 = Cfg::NB1, NB2 = Cfg::NB2;
#pragma unroll
    for (int m = 0; m < NB1; ++m) dft_br<R1, NB1, LO1, R1>(&re[m], &im[m]);
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

}  // namespace fsp

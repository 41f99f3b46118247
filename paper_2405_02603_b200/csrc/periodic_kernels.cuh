// periodic_kernels.cuh -- the z pass for a PERIODIC z direction at the cost the paper's step 1 implies (PAPER.md:67:
// only the non-periodic directions are doubled; reading R20).
//
// FSP_PARAM_PERIODIC works with the unchanged doubled-grid kernels because the folded table's spectrum has zero odd bins.
// Along z that wastes half of K3, the dominant kernel: the cyclic convolution of period Nz needs Nz-point transforms only,
//     y = IDFT_Nz( G_Nz . DFT_Nz(x) ),   G_Nz[j] = Ghat_2Nz[2j] / 2,
// and the 1/(2 Nz) folded into the stored spectrum is exactly (1/Nz)(1/2): the rows are used as they are, the even
// entries of either row layout (Ghat is even in kz).  No padding, no pruning:
// one pencil of Nz points per lane group of Fft2Cfg<Nz>, forward, times Ghat, inverse by IFFT(Y) = conj(FFT(conj Y)) on
// ONE copy of the transform code, in place in B2.  Same layout of B2 as K3 (the x and y passes are the doubled-grid ones).
#pragma once
#include <cuda_runtime.h>
#include "fft_warp.cuh"

namespace fsp {

template <int M>
struct ConvZPer {
    using Cfg = Fft2Cfg<M>;
    // (8 warps also where 16 points per lane would allow more: at Nz = 256 12 warps at 164 registers take 0.229 ms and
    // 16 at 128 registers 0.252 ms against 0.201 ms)
    static constexpr int T = Cfg::T, R = Cfg::R, G = 32 / T, WARPS = 8, ROW = M + 2;
    static constexpr size_t smem_bytes() { return sizeof(double2) * (size_t)(WARPS * G * Cfg::BUF); }
};

template <int M, bool NATURAL>
__global__ void __launch_bounds__(ConvZPer<M>::WARPS * 32, 1)
k_conv_z_periodic(double2* __restrict__ B2, const double* __restrict__ Gk, const double* __restrict__ lane_g, int Ny,
                  long ngroups, long npencils) {
    using Z = ConvZPer<M>;
    using Cfg = typename Z::Cfg;
    constexpr int R = Z::R, T = Z::T, G = Z::G, WARPS = Z::WARPS, NC = LaneTw<Cfg::R2>::NC, NB2 = Cfg::NB2;
    extern __shared__ double2 smzp[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane / T, t = lane % T;
    double2* buf = smzp + (warp * G + g) * Cfg::BUF;
    double cc[NB2][NC], tn[NB2][NC];
#pragma unroll
    for (int m = 0; m < NB2; ++m)
#pragma unroll
        for (int i = 0; i < NC; ++i) {
            cc[m][i] = lane_g[(t + T * m) * 2 * NC + i];
            tn[m][i] = lane_g[(t + T * m) * 2 * NC + NC + i];
        }
    const long ny2 = 2L * Ny;
    for (long grp = (long)blockIdx.x * WARPS + warp; grp < ngroups; grp += (long)gridDim.x * WARPS) {
        long pen = grp * G + g;   // = kx * 2 Ny + ky
        // (G divides the 2 Ny pencils of a plane unless G = 16: the last group may then be ragged)
        constexpr bool RAGGED = G > 8;
        bool valid = true;
        if constexpr (RAGGED) {
            valid = pen < npencils;
            if (!valid) pen = npencils - 1;
        }
        const long kx = pen / ny2;
        const int ky = (int)(pen - kx * ny2), qy = ky <= Ny ? ky : (int)ny2 - ky;
        double2* base = B2 + pen * M;
        const double* row = Gk + (kx * (Ny + 1) + qy) * Z::ROW;
        double vr[R], vi[R];
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const double2 v = base[t + T * i];
            vr[i] = v.x; vi[i] = v.y;
        }
        if constexpr (M <= 256) {   // L2 prefetch of this lane group's next pencil, M * 16 / 128 lines (measured: 256^3
                                    // 0.221 -> 0.201 ms; at Nz = 512 it costs 3 %, so not there)
            const long nxt = pen + (long)gridDim.x * WARPS * G;
            if (nxt < npencils) {
                const double2* nb = B2 + nxt * M;
#pragma unroll
                for (int e = 0; e < M / 8; e += T) asm volatile("prefetch.global.L2 [%0];" ::"l"(nb + (e + t) * 8));
            }
        }
#pragma unroll 1
        for (int pass = 0; pass < 2; ++pass) {
            fft2_forward_lc<Cfg>(vr, vi, t, buf, cc, tn);
            if (pass == 0) {   // Y = conj(Ghat X)
#pragma unroll
                for (int i = 0; i < R; ++i) {
                    const int kz = t + T * i;
                    // Ghat_2Nz[2 kz] = Ghat_2Nz[2 Nz - 2 kz]: entry min(2 kz, 2 Nz - 2 kz) of a natural-order row, entry
                    // min(kz, Nz - kz) of the E half of an [E | O] row (k_layout_spectrum_oct: E[m] = Ghat[2 m])
                    const int e = kz <= M - kz ? kz : M - kz;
                    const double gk = __ldg(row + (NATURAL ? 2 * e : e));
                    vr[i] *= gk; vi[i] *= -gk;
                }
            }
        }
#pragma unroll
        for (int i = 0; i < R; ++i)
            if (!RAGGED || valid) base[t + T * i] = make_double2(vr[i], -vi[i]);   // FFT(conj Y) = conj(y)
    }
}

}  // namespace fsp

// solve_kernels.cuh -- the five passes of one solve.
//
//   K1 fwd_x_r2c   rho[x][y][z] (real)          -> B1[kx<=Nx][y<Ny][z<Nz]   R2C along x, input-pruned
//   K2 fwd_y       B1                            -> B2[kx][ky<2Ny][z<Nz]     forward along y, input-pruned
//   K3 conv_z      B2 (in place)                 forward z (input-pruned) x Ghat, inverse z (output-pruned)
//   K4 inv_y       B2                            -> B1[kx][y<Ny][z<Nz]       inverse along y, output-pruned
//   K5 inv_x_c2r   B1                            -> phi[x][y][z] (real)      C2R along x, output-pruned
//
// Pruning identities used by every pass (N = mesh size along the axis, w = exp(-2 pi i/2N)):
//   zero-padded forward of length 2N with N non-zero inputs x[n]:
//       X[2j]   = FFT_N(x)[j],            X[2j+1] = FFT_N(x[n] w^n)[j]
//   inverse of length 2N of which only outputs n < N are kept:
//       y[n] = IFFT_N(Y[2j])[n] + conj(w^n) IFFT_N(Y[2j+1])[n]
// so the zero half of rho2 is never read and the discarded part of phi2
// is never computed or written.
//
// The x axis carries the real<->complex packing: z[n] = rho[2n] + i rho[2n+1] (adjacent x rows),
// a pruned length-Nx complex transform (two FFTs of length Nx/2), and the usual untangling
//       X'[k] = (A + B) - i w^k (A - B),   A = Z[k], B = conj(Z[Nx-k]),  k = 0..Nx    (X' = 2X)
// and its inverse  Z[k] = (A + B) + i conj(w^k) (A - B),  A = X[k], B = conj(X[Nx-k]).
// The factor 1/2 and hx hy hz/(8 Nx Ny Nz) live in Ghat.
#pragma once
#include <type_traits>
#include "fft_engine.cuh"
#include "fft_warp.cuh"

namespace fsp {

constexpr int kW = 8;  // complex columns per tile: 8 x 16 B = one 128-byte line per tile row

__device__ __forceinline__ void cmul(double& xr, double& xi, const double2 w) {
    const double a = xr * w.x - xi * w.y;
    xi = xr * w.y + xi * w.x;
    xr = a;
}
__device__ __forceinline__ void cmul_conj(double& xr, double& xi, const double2 w) {
    const double a = xr * w.x + xi * w.y;
    xi = xi * w.x - xr * w.y;
    xr = a;
}

// DER (field output, R18): the spectrum is additionally multiplied by -i k_d
// (k_d = kap.d * m', m' the signed mode number, zero at the Nyquist index; exactly one of kap.x/y/z is
// non-zero) and the result goes to `out` instead of back into B2, so that the forward data in B2 serve
// phi and all three components of E = -grad phi.
struct DerK { double x, y, z; int Nx; };

// x <- (-i c) x
__device__ __forceinline__ void mul_minus_i(double& xr, double& xi, const double c) { const double a = xr; xr = c * xi; xi = -c * a; }

__device__ __forceinline__ double signed_mode(int m, int N) { return m < N ? (double)m : (m == N ? 0.0 : (double)(m - 2 * N)); }

// copy the twiddle table exp(-2 pi i n/LTAB) into shared memory
template <int LTAB>
__device__ __forceinline__ void load_table(double2* __restrict__ Ws, const double2* __restrict__ Wg) {
    for (int n = threadIdx.x; n < LTAB; n += blockDim.x) Ws[n] = Wg[n];
}

// tiles per CTA so that a CTA has at least 128 threads
template <class Cfg> struct TileGroups { static constexpr int G = (kW * Cfg::T >= 128) ? 1 : 128 / (kW * Cfg::T); };

// ====================================================================================== K2: fwd_y
// grid: ceil(ntiles / G) CTAs of G*kW*T threads; tile = (kx, z-bundle of kW columns).
template <int M>
__global__ void __launch_bounds__(TileGroups<FftCfg<M>>::G* kW* FftCfg<M>::T)
k_fwd_y(const double2* __restrict__ B1, double2* __restrict__ B2, const double2* __restrict__ Wg,
        int Nz, long ntiles) {
    using Cfg = FftCfg<M>;
    constexpr int R = Cfg::R, T = Cfg::T, G = TileGroups<Cfg>::G, LTAB = 2 * M;
    extern __shared__ double2 smem[];
    double2* Ws = smem;                 // LTAB
    double2* xb = smem + LTAB;          // G * M * kW
    load_table<LTAB>(Ws, Wg);
    const int tid = threadIdx.x;
    const int g = tid / (kW * T), lt = tid % (kW * T);
    const int c = lt % kW, t = lt / kW;
    double2* buf = xb + g * (M * kW) + c;
    const int nzb = Nz / kW;
    __syncthreads();  // table ready
    // persistent CTAs: tile groups blockIdx.x, blockIdx.x + gridDim.x, ...; the next group's rows are
    // prefetched into L2 while this one is transformed
    for (long tile0 = (long)blockIdx.x * G; tile0 < ntiles; tile0 += (long)gridDim.x * G) {
        const long tile = tile0 + g;
        const bool valid = tile < ntiles;
        const long kx = valid ? tile / nzb : 0;
        const int zb = valid ? (int)(tile % nzb) : 0;
        const double2* in = B1 + (kx * M) * (long)Nz + zb * kW + c;
        double2* out = B2 + (kx * 2 * M) * (long)Nz + zb * kW + c;

        double xr[R], xi[R], vr[R], vi[R];
#pragma unroll
        for (int i = 0; i < R; ++i) {
            double2 v = valid ? in[(long)(t + T * i) * Nz] : make_double2(0.0, 0.0);
            xr[i] = v.x; xi[i] = v.y;
        }
        {
            const long tn = tile + (long)gridDim.x * G;
            if (c == 0 && tn < ntiles) {
                const double2* nin = B1 + ((tn / nzb) * M) * (long)Nz + (tn % nzb) * kW;
#pragma unroll
                for (int i = 0; i < R; ++i) asm volatile("prefetch.global.L2 [%0];" ::"l"(nin + (long)(t + T * i) * Nz));
            }
        }
        // even outputs
#pragma unroll
        for (int i = 0; i < R; ++i) { vr[i] = xr[i]; vi[i] = xi[i]; }
        fft_forward<Cfg, kW, LTAB>(vr, vi, t, buf, Ws);
        if (valid) {
#pragma unroll
            for (int i = 0; i < R; ++i) out[(long)(2 * (t + T * i)) * Nz] = make_double2(vr[i], vi[i]);
        }
        // odd outputs
#pragma unroll
        for (int i = 0; i < R; ++i) { cmul(xr[i], xi[i], Ws[t + T * i]); }
        fft_forward<Cfg, kW, LTAB>(xr, xi, t, buf, Ws);
        if (valid) {
#pragma unroll
            for (int i = 0; i < R; ++i) out[(long)(2 * (t + T * i) + 1) * Nz] = make_double2(xr[i], xi[i]);
        }
    }
}

// ================================================================================= K2 (v2): fwd_y_t
// Tile kernel: one CTA = two groups of kW*T threads, group 0 computes the even
// outputs of the pruned transform, group 1 the odd ones (input times w^n first).  The tile
// [M rows][kW columns] arrives by TMA (tensor map over B1 viewed as [kx][y][2 Nz doubles]) into X; both
// groups copy it to registers, after which X is handed back to the TMA for the NEXT tile while this one
// is transformed: global-load latency never reaches the FFT.  Results go straight from registers to
// global memory, four full 128-byte lines per warp instruction.
template <int M>
struct TileY {
    using Cfg = Fft2Cfg<M>;
    static constexpr int T = Cfg::T, R = Cfg::R;
    static constexpr int KW = (M >= 1024) ? 4 : kW;   // columns per tile: 1024 rows x 8 columns would not fit shared memory
    static constexpr int GT = KW * T;             // threads per group
    static constexpr int THREADS = 2 * GT;
    static constexpr int NC = LaneTw<Cfg::R2>::NC;
    static constexpr int MINB = (M >= 512) ? 1 : (M >= 256 ? 2 : 4);
    static constexpr int BOXR = M < 256 ? M : 256;   // rows per TMA box (box dimensions are limited to 256)
    // [mbarriers: 128 B][X: M*kW][E: 2 groups x M*kW][wp: M]
    static constexpr size_t smem_bytes() { return 128 + sizeof(double2) * (size_t)(3 * M * KW + M); }
};

template <int M>
__global__ void __launch_bounds__(TileY<M>::THREADS, TileY<M>::MINB)
k_fwd_y_t(const __grid_constant__ CUtensorMap tmB1, double2* __restrict__ B2, const double* __restrict__ lane_g,
          const double2* __restrict__ wp_g, int Nz, int kx0, long ntiles) {
    using Y = TileY<M>;
    using Cfg = typename Y::Cfg;
    constexpr int R = Y::R, T = Y::T, GT = Y::GT, NC = Y::NC, NB2 = Cfg::NB2, KW = Y::KW;
    extern __shared__ __align__(128) unsigned char smraw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smraw);
    double2* X = reinterpret_cast<double2*>(smraw + 128);
    double2* E = X + M * KW;
    double2* wp = E + 2 * M * KW;
    const int tid = threadIdx.x;
    const int grp = tid / GT, gt = tid % GT, c = gt % KW, t = gt / KW;
    for (int n = tid; n < M; n += Y::THREADS) wp[n] = wp_g[n];
    double cc[NB2][NC], tn[NB2][NC];
#pragma unroll
    for (int m = 0; m < NB2; ++m)
#pragma unroll
        for (int i = 0; i < NC; ++i) {
            cc[m][i] = lane_g[(t + T * m) * 2 * NC + i];
            tn[m][i] = lane_g[(t + T * m) * 2 * NC + NC + i];
        }
    if (tid == 0) { mbar_init(full, 1); mbar_fence_init(); }
    __syncthreads();
    const int nzb = Nz / KW;
    auto issue = [&](long tile) {   // one thread: arm the barrier, then one TMA per box of rows
        const int kx = (int)(tile / nzb), zb = (int)(tile % nzb);
        mbar_arrive_expect_tx(full, (uint32_t)(M * KW * sizeof(double2)));
#pragma unroll
        for (int r0 = 0; r0 < M; r0 += Y::BOXR) tma_load_3d(X + r0 * KW, &tmB1, full, zb * KW * 2, r0, kx0 + kx);
    };
    long tile = blockIdx.x;
    if (tid == 0 && tile < ntiles) issue(tile);
    uint32_t parity = 0;
    double2* Ec = E + grp * (M * KW) + c;
    for (; tile < ntiles; tile += gridDim.x) {
        const long kx = tile / nzb;
        const int zb = (int)(tile % nzb);
        double vr[R], vi[R];
        mbar_wait(full, parity);
        parity ^= 1;
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const double2 v = X[(t + T * i) * KW + c];
            vr[i] = v.x; vi[i] = v.y;
        }
        __syncthreads();   // every thread holds its part of the tile: X may be refilled
        if (tid == 0 && tile + gridDim.x < ntiles) issue(tile + gridDim.x);
        if (grp) {
#pragma unroll
            for (int i = 0; i < R; ++i) cmul(vr[i], vi[i], wp[t + T * i]);
        }
        fft2_forward_tile<Cfg, KW>(vr, vi, t, Ec, 1 + grp, cc, tn);
        double2* out = B2 + ((kx * 2 * M + grp) * (long)Nz + zb * KW + c);
#pragma unroll
        for (int i = 0; i < R; ++i) out[(long)(2 * (t + T * i)) * Nz] = make_double2(vr[i], vi[i]);
    }
}

// ================================================================================= K2 (v3): fwd_y_f
// The tile kernel with ONE group per tile that transforms the whole zero-padded column of M2 = 2 Ny points (as
// k_conv_z_f does along z): the tile is read from shared memory once instead of twice, there is no pre-twiddle
// x[n] w^n and no twiddle table; the first radix-2 level of stage 1 is a register copy made while loading.
// Ny = 512: M2 = 1024 = 32 x 32, 8 columns x 32 lanes = 256 threads, 32 points per lane.
template <int M2>
struct TileYF {
    using Cfg = Fft2Cfg<M2>;
    static constexpr int M = M2 / 2;                 // Ny
    static constexpr int T = Cfg::T, R = Cfg::R, KW = kW;
    static constexpr int THREADS = KW * T;
    static constexpr int NC = LaneTw<Cfg::R2>::NC;
    static constexpr int BOXR = M < 256 ? M : 256;
    static_assert(Cfg::NB1 == 1 && Cfg::NB2 == 1, "one butterfly per lane and stage");
    // [mbarriers: 128 B][X: M*KW][E: M2*KW]
    static constexpr size_t smem_bytes() { return 128 + sizeof(double2) * (size_t)(M * KW + M2 * KW); }
};

template <int M2>
__global__ void __launch_bounds__(TileYF<M2>::THREADS, 1)
k_fwd_y_f(const __grid_constant__ CUtensorMap tmB1, double2* __restrict__ B2, const double* __restrict__ lane_g,
          int Nz, int kx0, long ntiles) {
    using Y = TileYF<M2>;
    using Cfg = typename Y::Cfg;
    constexpr int R = Y::R, T = Y::T, NC = Y::NC, KW = Y::KW, M = Y::M, H = R / 2;
    extern __shared__ __align__(128) unsigned char smraw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smraw);
    double2* X = reinterpret_cast<double2*>(smraw + 128);
    double2* E = X + M * KW;
    const int tid = threadIdx.x;
    const int c = tid % KW, t = tid / KW;
    double cc[1][NC], tn[1][NC];
#pragma unroll
    for (int i = 0; i < NC; ++i) {
        cc[0][i] = lane_g[t * 2 * NC + i];
        tn[0][i] = lane_g[t * 2 * NC + NC + i];
    }
    if (tid == 0) { mbar_init(full, 1); mbar_fence_init(); }
    __syncthreads();
    const int nzb = Nz / KW;
    auto issue = [&](long tile) {   // one thread: arm the barrier, then one TMA per box of rows
        const int kx = (int)(tile / nzb), zb = (int)(tile % nzb);
        mbar_arrive_expect_tx(full, (uint32_t)(M * KW * sizeof(double2)));
#pragma unroll
        for (int r0 = 0; r0 < M; r0 += Y::BOXR) tma_load_3d(X + r0 * KW, &tmB1, full, zb * KW * 2, r0, kx0 + kx);
    };
    long tile = blockIdx.x;
    if (tid == 0 && tile < ntiles) issue(tile);
    uint32_t parity = 0;
    double2* Ec = E + c;
    for (; tile < ntiles; tile += gridDim.x) {
        const long kx = tile / nzb;
        const int zb = (int)(tile % nzb);
        double vr[R], vi[R];
        mbar_wait(full, parity);
        parity ^= 1;
#pragma unroll
        for (int i = 0; i < H; ++i) {   // rows t + T i < Ny; the zero half: (x_i, 0) -> (x_i, x_i)
            const double2 v = X[(t + T * i) * KW + c];
            vr[i] = v.x; vi[i] = v.y;
            vr[i + H] = v.x; vi[i + H] = v.y;
        }
        __syncthreads();   // every thread holds its part of the tile: X may be refilled
        if (tid == 0 && tile + gridDim.x < ntiles) issue(tile + gridDim.x);
        fft2_forward_tile<Cfg, KW, 4>(vr, vi, t, Ec, 1, cc, tn);
        double2* out = B2 + ((kx * M2) * (long)Nz + zb * KW + c);
#pragma unroll
        for (int i = 0; i < R; ++i) out[(long)(t + T * i) * Nz] = make_double2(vr[i], vi[i]);
    }
}

// ====================================================================================== K4: inv_y
// DER: input row ky is multiplied by -i kder m'(ky) first (E_y of the field output, see DerK)
template <int M, bool DER = false>
__global__ void __launch_bounds__(TileGroups<FftCfg<M>>::G* kW* FftCfg<M>::T)
k_inv_y(const double2* __restrict__ B2, double2* __restrict__ B1, const double2* __restrict__ Wg,
        int Nz, long ntiles, const double kder) {
    using Cfg = FftCfg<M>;
    constexpr int R = Cfg::R, T = Cfg::T, G = TileGroups<Cfg>::G, LTAB = 2 * M;
    extern __shared__ double2 smem[];
    double2* Ws = smem;
    double2* xb = smem + LTAB;
    load_table<LTAB>(Ws, Wg);
    const int tid = threadIdx.x;
    const int g = tid / (kW * T), lt = tid % (kW * T);
    const int c = lt % kW, t = lt / kW;
    double2* buf = xb + g * (M * kW) + c;
    const int nzb = Nz / kW;
    __syncthreads();  // table ready
    for (long tile0 = (long)blockIdx.x * G; tile0 < ntiles; tile0 += (long)gridDim.x * G) {
        const long tile = tile0 + g;
        const bool valid = tile < ntiles;
        const long kx = valid ? tile / nzb : 0;
        const int zb = valid ? (int)(tile % nzb) : 0;
        const double2* in = B2 + (kx * 2 * M) * (long)Nz + zb * kW + c;
        double2* out = B1 + (kx * M) * (long)Nz + zb * kW + c;

        double er[R], ei[R], qr[R], qi[R];
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const long row = 2 * (t + T * i);
            double2 a = valid ? in[row * Nz] : make_double2(0.0, 0.0);
            double2 b = valid ? in[(row + 1) * Nz] : make_double2(0.0, 0.0);
            er[i] = a.x; ei[i] = a.y; qr[i] = b.x; qi[i] = b.y;
            if constexpr (DER) {
                mul_minus_i(er[i], ei[i], kder * signed_mode((int)row, M));
                mul_minus_i(qr[i], qi[i], kder * signed_mode((int)row + 1, M));
            }
        }
        {
            const long tn = tile + (long)gridDim.x * G;
            if (c == 0 && tn < ntiles) {
                const double2* nin = B2 + ((tn / nzb) * 2 * M) * (long)Nz + (tn % nzb) * kW;
#pragma unroll
                for (int i = 0; i < 2 * R; ++i) asm volatile("prefetch.global.L2 [%0];" ::"l"(nin + (long)(2 * t + 2 * T * (i >> 1) + (i & 1)) * Nz));
            }
        }
        fft_inverse<Cfg, kW, LTAB>(qr, qi, t, buf, Ws);
#pragma unroll
        for (int i = 0; i < R; ++i) cmul_conj(qr[i], qi[i], Ws[t + T * i]);
        fft_inverse<Cfg, kW, LTAB>(er, ei, t, buf, Ws);
        if (valid) {
#pragma unroll
            for (int i = 0; i < R; ++i)
                out[(long)(t + T * i) * Nz] = make_double2(er[i] + qr[i], ei[i] + qi[i]);
        }
    }
}

// ================================================================================= K4 (v2): inv_y_t
// Tile kernel, mirror image of k_fwd_y_t: group 0 inverse-transforms the even rows of the tile
// [2M rows][kW columns] of B2, group 1 the odd rows; then y[n] = y_e[n] + conj(w^n) y_o[n] for n < M.
// B2 is seen through a 4-D tensor map [plane][j][parity][2 Nz doubles], so that each group's TMA box
// holds the rows of one parity only.  Each group's buffer X_g receives the tile and then serves as the
// group's exchange buffer (same [position][kW] layout); once the exchange has been read back the buffer
// is handed to the TMA for the next tile (whose lines were prefetched into L2 when this tile started).
// The halves of y_e / y_o that the other group finishes travel through C.
template <int M>
struct TileYI {
    using Cfg = Fft2Cfg<M>;
    static constexpr int T = Cfg::T, R = Cfg::R;
    static constexpr int KW = (M >= 1024) ? 4 : kW;
    static constexpr int GT = KW * T, THREADS = 2 * GT;
    static constexpr int NC = LaneTw<Cfg::R2>::NC;
    static constexpr int MINB = (M >= 512) ? 1 : (M >= 256 ? 2 : 4);
    static constexpr int BOXR = M < 256 ? M : 256;
    // [mbarriers: 128 B][X: 2 groups x M*kW][C: 2 groups x (M/2)*kW][wp: M]
    static constexpr size_t smem_bytes() { return 128 + sizeof(double2) * (size_t)(3 * M * KW + M); }
};

template <int M, bool DER = false>
__global__ void __launch_bounds__(TileYI<M>::THREADS, TileYI<M>::MINB)
k_inv_y_t(const __grid_constant__ CUtensorMap tmB2, double2* __restrict__ B1, const double* __restrict__ lane_g,
          const double2* __restrict__ wp_g, int Nz, long ntiles, const double kder) {
    using Y = TileYI<M>;
    using Cfg = typename Y::Cfg;
    constexpr int R = Y::R, T = Y::T, GT = Y::GT, NC = Y::NC, NB2 = Cfg::NB2, H = R / 2, KW = Y::KW;
    extern __shared__ __align__(128) unsigned char smraw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smraw);   // full[0], full[1]
    double2* X = reinterpret_cast<double2*>(smraw + 128);
    double2* C = X + 2 * M * KW;
    double2* wp = C + M * KW;
    const int tid = threadIdx.x;
    const int grp = tid / GT, gt = tid % GT, c = gt % KW, t = gt / KW;
    for (int n = tid; n < M; n += Y::THREADS) wp[n] = wp_g[n];
    double cc[NB2][NC], tn[NB2][NC];
#pragma unroll
    for (int m = 0; m < NB2; ++m)
#pragma unroll
        for (int i = 0; i < NC; ++i) {
            cc[m][i] = lane_g[(t + T * m) * 2 * NC + i];
            tn[m][i] = lane_g[(t + T * m) * 2 * NC + NC + i];
        }
    if (tid == 0) { mbar_init(&full[0], 1); mbar_init(&full[1], 1); mbar_fence_init(); }
    __syncthreads();
    const int nzb = Nz / KW;
    double2* Xg = X + grp * (M * KW);
    auto issue = [&](long tile) {   // one thread of the group: this group's rows of the tile
        const int kx = (int)(tile / nzb), zb = (int)(tile % nzb);
        mbar_arrive_expect_tx(&full[grp], (uint32_t)(M * KW * sizeof(double2)));
#pragma unroll
        for (int r0 = 0; r0 < M; r0 += Y::BOXR) tma_load_4d(Xg + r0 * KW, &tmB2, &full[grp], zb * KW * 2, grp, r0, kx);
    };
    auto prefetch = [&](long tile) {
        const int kx = (int)(tile / nzb), zb = (int)(tile % nzb);
#pragma unroll
        for (int r0 = 0; r0 < M; r0 += Y::BOXR) tma_prefetch_4d(&tmB2, zb * KW * 2, grp, r0, kx);
    };
    long tile = blockIdx.x;
    if (gt == 0 && tile < ntiles) issue(tile);
    uint32_t parity = 0;
    double2* Ec = Xg + c;
    double2* Cmine = C + grp * (M / 2 * KW) + c;          // what this group gives away
    double2* Ctheirs = C + (grp ^ 1) * (M / 2 * KW) + c;  // what it receives
    for (; tile < ntiles; tile += gridDim.x) {
        const long kx = tile / nzb;
        const int zb = (int)(tile % nzb);
        const bool more = tile + gridDim.x < ntiles;
        if (gt == 0 && more) prefetch(tile + gridDim.x);
        double vr[R], vi[R];
        mbar_wait(&full[grp], parity);
        parity ^= 1;
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const double2 v = Ec[(t + T * i) * KW];
            vr[i] = v.x; vi[i] = v.y;
            if constexpr (DER) mul_minus_i(vr[i], vi[i], kder * signed_mode(2 * (t + T * i) + grp, M));
        }
        // inverse transform = forward transform with the roles of re and im swapped; the first barrier
        // inside also separates the reads of X_g above from its reuse as exchange buffer
        fft2_forward_tile<Cfg, KW>(vi, vr, t, Ec, 1 + grp, cc, tn);
        bar_sync(1 + grp, GT);   // exchange read back by the whole group: X_g is free
        if (gt == 0 && more) { fence_proxy_async(); issue(tile + gridDim.x); }
        __syncthreads();         // C of the previous tile has been consumed by both groups
#pragma unroll
        for (int i = 0; i < H; ++i) {
            const int s = grp ? i : i + H;    // group 1 gives away y_o[n], i < H; group 0 gives y_e[n], i >= H
            Cmine[(t + T * i) * KW] = make_double2(vr[s], vi[s]);
        }
        __syncthreads();
        double2* out = B1 + ((kx * M) * (long)Nz + zb * KW + c);
#pragma unroll
        for (int i = 0; i < H; ++i) {
            const double2 pv = Ctheirs[(t + T * i) * KW];
            const int o = grp ? i + H : i;
            const double er = grp ? pv.x : vr[i], ei = grp ? pv.y : vi[i];                 // y_e[n]
            const double qr = grp ? vr[i + H] : pv.x, qi = grp ? vi[i + H] : pv.y;         // y_o[n]
            const double2 w = wp[t + T * o];
            // y = y_e + conj(w) y_o
            const double yr = fma(w.y, qi, fma(w.x, qr, er));
            const double yi = fma(-w.y, qr, fma(w.x, qi, ei));
            out[(long)(t + T * o) * Nz] = make_double2(yr, yi);
        }
    }
}

// ============================================================ K3 for any supported Nz (3 * 2^k, 5 * 2^k): conv_z_g
// CTA-level kernel on the register engine of fft_engine.cuh (any radix mix), used where the warp-level kernels do
// not apply (Nz not a power of two).  Tile = kW pencils that follow one another in memory (pencil
// q = (kx, ky), M contiguous points each); thread (c, t) = (pencil of the tile, lane of the pencil), c fastest, so
// that the exchange buffer [position][kW] is conflict free.  Per pencil: both half-spectrum branches one after the
// other (even: FFT_M(x); odd: FFT_M(x w^n)), times the octant spectrum row [E | O], inverse, y = y_e + conj(w^n) y_o.
template <int M, bool DER = false>
__global__ void __launch_bounds__(TileGroups<FftCfg<M>>::G* kW* FftCfg<M>::T)
k_conv_z_g(double2* __restrict__ B2, const double* __restrict__ Gk, const double2* __restrict__ Wg, int Ny,
           long npencils, double2* __restrict__ out, const DerK kap) {
    using Cfg = FftCfg<M>;
    constexpr int R = Cfg::R, T = Cfg::T, G = TileGroups<Cfg>::G, LTAB = 2 * M, ROW = M + 2;
    extern __shared__ double2 smem[];
    double2* Ws = smem;                 // LTAB: exp(-2 pi i n / 2M)
    double2* xb = smem + LTAB;          // G * M * kW
    load_table<LTAB>(Ws, Wg);
    const int tid = threadIdx.x;
    const int g = tid / (kW * T), lt = tid % (kW * T);
    const int c = lt % kW, t = lt / kW;
    double2* buf = xb + g * (M * kW) + c;
    const int ny2 = 2 * Ny;
    __syncthreads();
    for (long tile0 = (long)blockIdx.x * G; tile0 * kW < npencils; tile0 += (long)gridDim.x * G) {
        const long q = (tile0 + g) * kW + c;
        const bool valid = q < npencils;
        const int kx = valid ? (int)(q / ny2) : 0, ky = valid ? (int)(q % ny2) : 0;
        const int qy = ky <= Ny ? ky : ny2 - ky;
        double2* base = B2 + (valid ? q : 0) * M;
        double2* obase = DER ? out + (valid ? q : 0) * M : base;
        const double* grow = Gk + ((long)kx * (Ny + 1) + qy) * ROW;
        double fp = 0.0;
        if constexpr (DER) fp = kap.x * signed_mode(kx, kap.Nx) + kap.y * signed_mode(ky, Ny);
        double xr[R], xi[R], vr[R], vi[R];
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const double2 v = valid ? base[t + T * i] : make_double2(0.0, 0.0);
            xr[i] = v.x; xi[i] = v.y; vr[i] = v.x; vi[i] = v.y;
        }
        // even branch: Y_e[j] = Ghat[2j] FFT_M(x)[j], y_e = IFFT_M(Y_e) (kept in vr, vi)
        fft_forward<Cfg, kW, LTAB>(vr, vi, t, buf, Ws);
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const int j = t + T * i;
            double gk = __ldg(grow + (j <= M - j ? j : M - j));
            if constexpr (DER) gk *= fp + kap.z * signed_mode(2 * j, M);
            vr[i] *= gk; vi[i] *= gk;
        }
        fft_inverse<Cfg, kW, LTAB>(vr, vi, t, buf, Ws);
        // odd branch: x[n] w^n, Y_o[j] = Ghat[2j+1] FFT_M(.)[j], y_o = IFFT_M(Y_o)
#pragma unroll
        for (int i = 0; i < R; ++i) cmul(xr[i], xi[i], Ws[t + T * i]);
        fft_forward<Cfg, kW, LTAB>(xr, xi, t, buf, Ws);
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const int j = t + T * i;
            double gk = __ldg(grow + M / 2 + 1 + (j <= M - 1 - j ? j : M - 1 - j));
            if constexpr (DER) gk *= fp + kap.z * signed_mode(2 * j + 1, M);
            xr[i] *= gk; xi[i] *= gk;
        }
        fft_inverse<Cfg, kW, LTAB>(xr, xi, t, buf, Ws);
        if (valid) {
#pragma unroll
            for (int i = 0; i < R; ++i) {
                cmul_conj(xr[i], xi[i], Ws[t + T * i]);
                const double yr = vr[i] + xr[i], yi = vi[i] + xi[i];
                obase[t + T * i] = DER ? make_double2(yi, -yr) : make_double2(yr, yi);   // DER: -i y
            }
        }
    }
}

// ================================================ K3 for Nz = 3 * 2^k, 5 * 2^k with a kernel of length 2 Nz: conv_z_g2
// The same tile scheme as k_conv_z_g, but each pencil is transformed as ONE zero-padded sequence of M2 = 2 Nz points
// (forward, times Ghat in natural order, inverse, first half kept) instead of two half-length branches each way:
// one register set instead of two (no spills at R = 24), no pre-twiddle, no final sum.  The zero half is fed to the
// first stage as zeros and the discarded half is computed and dropped (the engine's stages are generic; the pruned
// first / last radix-2 levels of k_conv_z_f do not exist for these radices).
template <int M2, bool DER = false>
__global__ void __launch_bounds__(TileGroups<FftCfg<M2>>::G* kW* FftCfg<M2>::T)
k_conv_z_g2(double2* __restrict__ B2, const double* __restrict__ Gk, const double2* __restrict__ Wg, int Ny,
            long npencils, double2* __restrict__ out, const DerK kap) {
    using Cfg = FftCfg<M2>;
    constexpr int R = Cfg::R, T = Cfg::T, G = TileGroups<Cfg>::G, LTAB = M2, M = M2 / 2, ROW = M + 2;
    extern __shared__ double2 smem[];
    double2* Ws = smem;                 // LTAB: exp(-2 pi i n / M2)
    double2* xb = smem + LTAB;          // G * M2 * kW
    load_table<LTAB>(Ws, Wg);
    const int tid = threadIdx.x;
    const int g = tid / (kW * T), lt = tid % (kW * T);
    const int c = lt % kW, t = lt / kW;
    double2* buf = xb + g * (M2 * kW) + c;
    const int ny2 = 2 * Ny;
    __syncthreads();
    for (long tile0 = (long)blockIdx.x * G; tile0 * kW < npencils; tile0 += (long)gridDim.x * G) {
        const long q = (tile0 + g) * kW + c;
        const bool valid = q < npencils;
        const int kx = valid ? (int)(q / ny2) : 0, ky = valid ? (int)(q % ny2) : 0;
        const int qy = ky <= Ny ? ky : ny2 - ky;
        double2* base = B2 + (valid ? q : 0) * M;
        double2* obase = DER ? out + (valid ? q : 0) * M : base;
        const double* grow = Gk + ((long)kx * (Ny + 1) + qy) * ROW;
        double fp = 0.0;
        if constexpr (DER) fp = kap.x * signed_mode(kx, kap.Nx) + kap.y * signed_mode(ky, Ny);
        double vr[R], vi[R];
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const int n = t + T * i;
            const double2 v = (valid && n < M) ? base[n] : make_double2(0.0, 0.0);
            vr[i] = v.x; vi[i] = v.y;
        }
        fft_forward<Cfg, kW, LTAB>(vr, vi, t, buf, Ws);
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const int kz = t + T * i;
            double gk = __ldg(grow + (kz <= M ? kz : M2 - kz));
            if constexpr (DER) gk *= fp + kap.z * signed_mode(kz, M);
            vr[i] *= gk; vi[i] *= gk;
        }
        fft_inverse<Cfg, kW, LTAB>(vr, vi, t, buf, Ws);
        if (valid) {
#pragma unroll
            for (int i = 0; i < R; ++i) {
                const int n = t + T * i;
                if (n < M) obase[n] = DER ? make_double2(vi[i], -vr[i]) : make_double2(vr[i], vi[i]);   // DER: -i y
            }
        }
    }
}

// ============================================================================== K3 (v2): conv_z_w
// One pencil per group of 2T lanes of a warp: lanes with b = 0 run the even
// half-spectrum branch, lanes with b = 1 the odd one, each a two-stage single-exchange FFT of
// fft_warp.cuh over T lanes with R points per lane.  Both branches read the same x (one fetch,
// broadcast), read their half of the spectrum row (E or O), and the final sum y = y_e + conj(w^n) y_o
// is formed with one shuffle per value; each branch then stores half of the pencil.
//
// Spectrum layout Gk (k_layout_spectrum_oct): only the unique octant of the real, even spectrum is
// stored, row (kx, qy) = [ E[0..M/2] | O[0..M/2-1] | pad ], E[m] = Ghat[2m], O[m] = Ghat[2m+1], so
//     Ghat[kz = 2j]   = E[min(j, M - j)],      Ghat[kz = 2j+1] = O[min(j, M-1-j)],     row of ky = row of 2Ny-ky.
// Pencils are visited in the order ky = 0, 2Ny-1, 1, 2Ny-2, 2, ... so that the two pencils sharing a
// spectrum row are processed back to back by neighbouring warps (second read hits L2).
//
// Persistent warps: warp w of the grid handles pencil groups w, w + nwarps, ... (no CTA barrier after
// the tables are loaded).  The next group's x is prefetched into L2 while this one is transformed.
template <int M>
struct ConvZ {
    using Cfg = Fft2Cfg<M>;
    static constexpr int T = Cfg::T, R = Cfg::R;
    static constexpr int G = 16 / T;                 // pencils per warp at a time
    static constexpr int WARPS = 4;                  // warps per CTA
    static constexpr int ROW = M + 2;                // doubles per spectrum row (E: M/2+1, O: M/2, pad 1)
    static constexpr int NC = LaneTw<Cfg::R2>::NC;   // lane-constant twiddles per stage-2 butterfly
    // the spectrum row of the current pencil is staged in shared memory by a bulk async copy issued when
    // the pencil starts, so that its (HBM) latency is spent under the forward transform (only G == 1)
    static constexpr bool GSTAGE = (G == 1);
    static constexpr int GROW = GSTAGE ? ROW : 0;    // doubles of staging per warp
    // [wp: M double2][exchange: WARPS*2*G*BUF double2][G rows: WARPS*GROW doubles][mbarriers: WARPS]
    static constexpr size_t smem_bytes() {
        return sizeof(double2) * (size_t)(M + WARPS * 2 * G * Cfg::BUF) + sizeof(double) * (size_t)(WARPS * GROW) + 8 * WARPS;
    }
};

template <int M, bool DER = false>
__global__ void __launch_bounds__(ConvZ<M>::WARPS * 32, (M >= 512 ? 2 : 3))
k_conv_z_w(double2* __restrict__ B2, const double* __restrict__ Gk, const double* __restrict__ lane_g,
           const double2* __restrict__ wp_g, int Ny, long ngroups, double2* __restrict__ out, const DerK kap) {
    using Z = ConvZ<M>;
    using Cfg = typename Z::Cfg;
    constexpr int R = Z::R, T = Z::T, G = Z::G, WARPS = Z::WARPS, H = R / 2, NC = Z::NC, NB2 = Cfg::NB2;
    extern __shared__ double2 smem[];
    double2* wp = smem;          // M: w_2M^n, n < M
    for (int n = threadIdx.x; n < M; n += blockDim.x) wp[n] = wp_g[n];
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane / (2 * T), b = (lane / T) & 1, t = lane % T;
    double2* buf = smem + M + ((warp * G + g) * 2 + b) * Cfg::BUF;
    double* gst = reinterpret_cast<double*>(smem + M + WARPS * 2 * G * Cfg::BUF) + warp * Z::GROW;
    uint64_t* gbar = reinterpret_cast<uint64_t*>(reinterpret_cast<double*>(smem + M + WARPS * 2 * G * Cfg::BUF) + WARPS * Z::GROW) + warp;
    if (Z::GSTAGE && lane == 0) { mbar_init(gbar, 1); mbar_fence_init(); }
    __syncwarp();
    uint32_t gpar = 0;
    // stage-2 twiddles of this lane's butterflies j = t + T*m, kept in registers for the whole kernel
    double cc[NB2][NC], tn[NB2][NC];
#pragma unroll
    for (int m = 0; m < NB2; ++m)
#pragma unroll
        for (int i = 0; i < NC; ++i) {
            cc[m][i] = lane_g[(t + T * m) * 2 * NC + i];
            tn[m][i] = lane_g[(t + T * m) * 2 * NC + NC + i];
        }
    const int nwarps = gridDim.x * WARPS;
    const int ny2 = 2 * Ny;
    for (int grp = blockIdx.x * WARPS + warp; grp < (int)ngroups; grp += nwarps) {
        const int s = grp * G + g;                        // position in the visiting order
        const int kx = s / ny2;
        const int r = s - kx * ny2;
        const int ky = (r & 1) ? ny2 - ((r + 1) >> 1) : (r >> 1);
        const int qy = ky <= Ny ? ky : ny2 - ky;
        double2* base = B2 + ((long)kx * ny2 + ky) * M;
        double2* obase = DER ? out + ((long)kx * ny2 + ky) * M : base;
        double fp = 0.0;   // pencil-constant part of the derivative factor
        if constexpr (DER) fp = kap.x * signed_mode(kx, kap.Nx) + kap.y * signed_mode(ky, Ny);
        const double* grow = Gk + ((long)kx * (Ny + 1) + qy) * Z::ROW + (b ? M / 2 + 1 : 0);
        if constexpr (Z::GSTAGE) {
            // all lanes are past the previous pencil's reads of gst (the shuffles of the final combine)
            if (lane == 0) {
                mbar_arrive_expect_tx(gbar, Z::ROW * 8);
                bulk_load(gst, Gk + ((long)kx * (Ny + 1) + qy) * Z::ROW, Z::ROW * 8, gbar);
            }
        }

        double vr[R], vi[R];
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const double2 v = base[t + T * i];
            vr[i] = v.x; vi[i] = v.y;
        }
        {   // L2 prefetch of the next group's pencil(s): 16-byte elements, one 128-byte line per 8
            const int s2 = s + nwarps * G;
            if (s2 < (int)ngroups * G) {
                const int kx2 = s2 / ny2;
                const int r2 = s2 - kx2 * ny2;
                const int ky2 = (r2 & 1) ? ny2 - ((r2 + 1) >> 1) : (r2 >> 1);
                const double2* nb = B2 + ((long)kx2 * ny2 + ky2) * M;
                for (int e = (b * T + t) * 8; e < M; e += 2 * T * 8)
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(nb + e));
            }
        }
        if (b) {
#pragma unroll
            for (int i = 0; i < R; ++i) cmul(vr[i], vi[i], wp[t + T * i]);
        }
        // Two passes over ONE copy of the transform code: IFFT(Y) = conj(FFT(conj(Y))).
        // Pass 0 ends with Y = conj(Ghat * X).
#pragma unroll 1
        for (int pass = 0; pass < 2; ++pass) {
            fft2_forward_lc<Cfg>(vr, vi, t, buf, cc, tn);
            if (pass == 0) {
                const double* gsrc = grow;
                if constexpr (Z::GSTAGE) {
                    mbar_wait(gbar, gpar);
                    gpar ^= 1;
                    gsrc = gst + (b ? M / 2 + 1 : 0);
                }
                // row index min(j, M-b-j), j = t + T i: j for the first half of the registers, M-b-j for the
                // second (T R = M), i.e. compile-time offsets from two lane pointers
                const double* gA = gsrc + t;
                const double* gB = gsrc + (M - b - t);
#pragma unroll
                for (int i = 0; i < R; ++i) {
                    const int j = t + T * i;
                    const double gk = Z::GSTAGE ? (i < R / 2 ? gA[T * i] : gB[-T * i])
                                                : (i < R / 2 ? __ldg(gA + T * i) : __ldg(gB - T * i));
                    if constexpr (DER) {   // conj(-i f Ghat X) = f Ghat (X.im + i X.re)
                        const double cf = gk * (fp + kap.z * signed_mode(2 * j + b, M));
                        vr[i] *= cf; vi[i] *= -cf;   // the factor -i is applied to the final sum
                    } else {
                        vr[i] *= gk; vi[i] *= -gk;
                    }
                }
            }
        }
        // now v = FFT(conj(Ghat X)), i.e. IFFT(Ghat X) = conj(v) on each branch, and
        //     y[n] = y_e[n] + conj(w^n) y_o[n] = conj( v_e[n] + w^n v_o[n] ).
        // Branch 0 finishes n = t + T*i for i < R/2, branch 1 for i >= R/2: one exchange of the halves,
        // then 4 FMAs per value on every lane.
#pragma unroll
        for (int i = 0; i < H; ++i) {
            const double sr = b ? vr[i] : vr[i + H], si = b ? vi[i] : vi[i + H];
            const double pr = __shfl_xor_sync(0xffffffffu, sr, T), pi = __shfl_xor_sync(0xffffffffu, si, T);
            const int o = b ? i + H : i;
            const double ar = b ? pr : vr[i], ai = b ? pi : vi[i];            // v_e[n]
            const double qr = b ? vr[i + H] : pr, qi = b ? vi[i + H] : pi;    // v_o[n]
            // w^(n + M/2) = -i w^n: both branches read the same table entry (one broadcast access)
            const double2 w0 = wp[t + T * i];
            const double2 w = b ? make_double2(w0.y, -w0.x) : w0;
            const double zr = fma(-w.y, qi, fma(w.x, qr, ar));
            const double zi = fma(w.y, qr, fma(w.x, qi, ai));
            obase[t + T * o] = DER ? make_double2(-zi, -zr) : make_double2(zr, -zi);   // DER: -i y
        }
    }
}

// ========================================================================= K3 (v2, pairs): conv_z_p
// A pencil is handled by a PAIR of warps: warp 2q runs the even half-spectrum branch, warp 2q+1 the odd one,
// each for G = 32/T pencils at a time (T lanes per pencil: Nz = 1024 -> T = 32, one pencil per pair step;
// Nz = 512, 256 -> T = 16, two).  Compared with k_conv_z_w (both branches in the two halves of ONE warp)
// nothing is executed under a branch predicate: the pre-twiddle of the odd branch costs issue slots in the
// odd warps only, and the final sum needs no per-lane selects.  Everything else is the same: one copy of the
// transform code run twice, lane-constant stage-2 twiddles, octant spectrum with the row(s) staged by bulk
// async copies per pair step, the visiting order that lets two pencils share a spectrum row in L2.  The
// final sum y[n] = conj(v_e[n] + w^n v_o[n]) exchanges half of each branch's values through the (then free)
// exchange buffers, with a named barrier over the pair; each warp stores half of each pencil.
template <int M>
struct ConvZP {
    using Cfg = Fft2Cfg<M>;
    static constexpr int T = Cfg::T, R = Cfg::R;
    static constexpr int G = 32 / T;                       // pencils per warp
    static constexpr int PAIRS = (M <= 256) ? 6 : 4, WARPS = 2 * PAIRS;
    static constexpr int MINB = 1;
    static constexpr int ROW = M + 2;
    static constexpr int NC = LaneTw<Cfg::R2>::NC;
    // [wp: M double2][exchange: WARPS*G*BUF double2][G rows: PAIRS*G*ROW doubles][mbarriers: PAIRS]
    static constexpr size_t smem_bytes() {
        return sizeof(double2) * (size_t)(M + WARPS * G * Cfg::BUF) + sizeof(double) * (size_t)(PAIRS * G * ROW) + 8 * PAIRS;
    }
};

template <int M, bool DER = false>
__global__ void __launch_bounds__(ConvZP<M>::WARPS * 32, ConvZP<M>::MINB)
k_conv_z_p(double2* __restrict__ B2, const double* __restrict__ Gk, const double* __restrict__ lane_g,
           const double2* __restrict__ wp_g, int Ny, long nsteps, double2* __restrict__ out, const DerK kap) {
    using Z = ConvZP<M>;
    using Cfg = typename Z::Cfg;
    constexpr int R = Z::R, T = Z::T, G = Z::G, PAIRS = Z::PAIRS, WARPS = Z::WARPS, NC = Z::NC, NB2 = Cfg::NB2;
    extern __shared__ double2 smem[];
    double2* wp = smem;          // M: w_2M^n, n < M
    for (int n = threadIdx.x; n < M; n += blockDim.x) wp[n] = wp_g[n];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, q = warp >> 1, b = warp & 1;
    const int g = lane / T, t = lane % T;
    double2* buf = smem + M + (warp * G + g) * Cfg::BUF;
    double2* pbuf = smem + M + ((warp ^ 1) * G + g) * Cfg::BUF;          // the partner's buffer
    double* gall = reinterpret_cast<double*>(smem + M + WARPS * G * Cfg::BUF);
    double* gst = gall + (q * G + g) * Z::ROW;
    uint64_t* gbar = reinterpret_cast<uint64_t*>(gall + PAIRS * G * Z::ROW) + q;
    if (b == 0 && lane == 0) { mbar_init(gbar, 1); mbar_fence_init(); }
    __syncthreads();
    uint32_t gpar = 0;
    double cc[NB2][NC], tn[NB2][NC];
#pragma unroll
    for (int m = 0; m < NB2; ++m)
#pragma unroll
        for (int i = 0; i < NC; ++i) {
            cc[m][i] = lane_g[(t + T * m) * 2 * NC + i];
            tn[m][i] = lane_g[(t + T * m) * 2 * NC + NC + i];
        }
    const int npairs = gridDim.x * PAIRS;
    const int ny2 = 2 * Ny;
    auto locate = [&](int s_, int& kx_, int& ky_) {   // position in the visiting order -> (kx, ky)
        kx_ = s_ / ny2;
        const int r_ = s_ - kx_ * ny2;
        ky_ = (r_ & 1) ? ny2 - ((r_ + 1) >> 1) : (r_ >> 1);
    };
    for (int step = blockIdx.x * PAIRS + q; step < (int)nsteps; step += npairs) {
        int kx, ky;
        locate(step * G + g, kx, ky);
        const int qy = ky <= Ny ? ky : ny2 - ky;
        double2* base = B2 + ((long)kx * ny2 + ky) * M;
        double2* obase = DER ? out + ((long)kx * ny2 + ky) * M : base;
        double fp = 0.0;
        if constexpr (DER) fp = kap.x * signed_mode(kx, kap.Nx) + kap.y * signed_mode(ky, Ny);
        // both warps are past the previous step's reads of the staged rows (the pair barrier ending the combine)
        if (b == 0 && lane == 0) {
            mbar_arrive_expect_tx(gbar, G * Z::ROW * 8);
#pragma unroll
            for (int gg = 0; gg < G; ++gg) {
                int kx2, ky2;
                locate(step * G + gg, kx2, ky2);
                const int qy2 = ky2 <= Ny ? ky2 : ny2 - ky2;
                bulk_load(gall + (q * G + gg) * Z::ROW, Gk + ((long)kx2 * (Ny + 1) + qy2) * Z::ROW, Z::ROW * 8, gbar);
            }
        }
        (void)qy;
        double vr[R], vi[R];
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const double2 v = base[t + T * i];
            vr[i] = v.x; vi[i] = v.y;
        }
        {   // L2 prefetch of the pair's next pencils, half of the lines from each warp
            const int s2 = (step + npairs) * G + g;
            if (step + npairs < (int)nsteps) {
                int kx2, ky2;
                locate(s2, kx2, ky2);
                const double2* nb = B2 + ((long)kx2 * ny2 + ky2) * M;
                for (int e = (b * T + t) * 8; e < M; e += 2 * T * 8)
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(nb + e));
            }
        }
        if (b) {
#pragma unroll
            for (int i = 0; i < R; ++i) cmul(vr[i], vi[i], wp[t + T * i]);
        }
#pragma unroll 1
        for (int pass = 0; pass < 2; ++pass) {
            fft2_forward_lc<Cfg>(vr, vi, t, buf, cc, tn);
            if (pass == 0) {
                mbar_wait(gbar, gpar);
                gpar ^= 1;
                const double* gsrc = gst + (b ? M / 2 + 1 : 0);
                const double* gA = gsrc + t;
                const double* gB = gsrc + (M - b - t);
                const double fz0 = fp + kap.z * (double)(2 * t + b);   // DER only
                const bool nyq = (2 * t + b) == 0;                      // register R/2 of this lane is kz = M
#pragma unroll
                for (int i = 0; i < R; ++i) {
                    const double gk = i < R / 2 ? gA[T * i] : gB[-T * i];   // row index min(j, M-b-j), j = t + T i
                    if constexpr (DER) {
                        // signed mode of kz = 2 (t + T i) + b: kz for the first half of the registers, kz - 2M for
                        // the second (T R = M), zero at the Nyquist index kz = M: a lane constant plus a
                        // compile-time offset, no integer arithmetic per point
                        // (the factor -i itself is applied to the final sum: F^-1 is linear)
                        double cf = gk * fma(kap.z, (double)(i < R / 2 ? 2 * T * i : 2 * T * i - 2 * M), fz0);
                        if (i == R / 2) cf = nyq ? gk * fp : cf;
                        vr[i] *= cf; vi[i] *= -cf;
                    } else {
                        vr[i] *= gk; vi[i] *= -gk;
                    }
                }
            }
        }
        // v = FFT(conj(Ghat X)) on each branch; y[n] = conj(v_e[n] + w^n v_o[n]).  The odd warp paid for the
        // pre-twiddle (4 fp64 instructions per point), so the even warp forms the whole sum (4 per point) and
        // stores the pencil: the two warps of a pair carry the same fp64 load.
        if (b) {
            __syncwarp();   // this warp's exchange reads are complete: buf becomes the outbox
#pragma unroll
            for (int i = 0; i < R; ++i) buf[t + T * i] = make_double2(vr[i], vi[i]);
        }
        bar_sync(1 + q, 64);
        if (!b) {
#pragma unroll
            for (int i = 0; i < R; ++i) {
                const double2 pv = pbuf[t + T * i];   // v_o[n], n = t + T i
                const double2 w = wp[t + T * i];
                const double zr = fma(-w.y, pv.y, fma(w.x, pv.x, vr[i]));
                const double zi = fma(w.y, pv.x, fma(w.x, pv.y, vi[i]));
                obase[t + T * i] = DER ? make_double2(-zi, -zr) : make_double2(zr, -zi);   // DER: -i y
            }
        }
        bar_sync(1 + q, 64);   // the even warp has read the outbox (and both are done with the staged rows)
    }
}

// ====================================================================== K3 (v4, Nz = 256, 512): conv_z_f
// One lane group transforms the WHOLE zero-padded pencil of M2 = 2 Nz points (1024 = 32 x 32 over a warp at
// Nz = 512; 512 = 16 x 32 over a half-warp, two pencils per warp, at Nz = 256) with fft2_padded_pass: forward with
// the zero half pruned inside stage 1, times Ghat, inverse with the discarded half pruned inside stage 2.  Against
// the branch-pair kernels (k_conv_z_p, k_conv_z_w: two half-length transforms per direction) the pencil is read
// once, there is no pre-twiddle x[n] w^n, no final sum y_e + conj(w^n) y_o, no twiddle table and no hand-over
// between warps: 704 instead of 992 L1/shared-memory wavefronts per pencil, the same fp64 work.
// Spectrum rows: the unique octant in natural order (k_layout_spectrum_nat), Ghat[kz] = row[min(kz, M2 - kz)]: every
// read is a lane pointer plus a compile-time offset.  Rows are staged by bulk async copies (one mbarrier per warp);
// visiting order as in k_conv_z_w (two pencils sharing a row run back to back).  Persistent warps, no CTA barrier.
template <int M2>
struct ConvZF {
    using Cfg = Fft2Cfg<M2>;
    static constexpr int M = M2 / 2;                       // Nz
    static constexpr int T = Cfg::T, R = Cfg::R;
    static constexpr int G = 32 / T;                       // pencils per warp
#ifndef FSP_ZF_WARPS
#define FSP_ZF_WARPS 8
#endif
    static constexpr int WARPS = FSP_ZF_WARPS;             // 8 warps at <= 255 registers (warps are allocated in fours:
                                                           // the next step, 12, leaves 168 registers and spills)
    static constexpr int ROW = M + 2;                      // doubles per spectrum row: Ghat[0..M], one pad
    static constexpr int NC = LaneTw<Cfg::R2>::NC;
    // [exchange: WARPS*G*BUF double2][G rows: WARPS*G*ROW doubles][mbarriers: WARPS]
    static constexpr size_t smem_bytes() {
        return sizeof(double2) * (size_t)(WARPS * G * Cfg::BUF) + sizeof(double) * (size_t)(WARPS * G * ROW) + 8 * WARPS;
    }
};

template <int M2, bool DER = false>
__global__ void __launch_bounds__(ConvZF<M2>::WARPS * 32, 1)
k_conv_z_f(double2* __restrict__ B2, const double* __restrict__ Gk, const double* __restrict__ lane_g, int Ny,
           long ngroups, double2* __restrict__ out, const DerK kap) {
    using Z = ConvZF<M2>;
    using Cfg = typename Z::Cfg;
    constexpr int M = Z::M, R = Z::R, T = Z::T, G = Z::G, WARPS = Z::WARPS, NC = Z::NC, H = R / 2;
    extern __shared__ double2 smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane / T, t = lane % T;
    double2* buf = smem + (warp * G + g) * Cfg::BUF;
    double* gall = reinterpret_cast<double*>(smem + WARPS * G * Cfg::BUF);
    double* gst = gall + (warp * G + g) * Z::ROW;
    uint64_t* gbar = reinterpret_cast<uint64_t*>(gall + WARPS * G * Z::ROW) + warp;
    if (lane == 0) { mbar_init(gbar, 1); mbar_fence_init(); }
    __syncwarp();
    uint32_t gpar = 0;
    double cc[NC], tn[NC];   // stage-2 twiddles of this lane's butterfly j = t, in registers for the whole kernel
#pragma unroll
    for (int i = 0; i < NC; ++i) {
        cc[i] = lane_g[t * 2 * NC + i];
        tn[i] = lane_g[t * 2 * NC + NC + i];
    }
    // Ghat[kz], kz = t + T i: the row entry min(kz, M2 - kz); rows are in natural order (k_layout_spectrum_nat), so a
    // lane group reads T consecutive doubles per instruction (no bank conflicts)
    const double* gA = gst + t;
    const double* gB = gst + (M2 - t);
    const int nwarps = gridDim.x * WARPS;
    const int ny2 = 2 * Ny;
    auto locate = [&](int s_, int& kx_, int& ky_) {   // position in the visiting order -> (kx, ky)
        kx_ = s_ / ny2;
        const int r_ = s_ - kx_ * ny2;
        ky_ = (r_ & 1) ? ny2 - ((r_ + 1) >> 1) : (r_ >> 1);
    };
    for (int grp = blockIdx.x * WARPS + warp; grp < (int)ngroups; grp += nwarps) {
        int kx, ky;
        locate(grp * G + g, kx, ky);
        double2* base = B2 + ((long)kx * ny2 + ky) * M;
        double2* obase = DER ? out + ((long)kx * ny2 + ky) * M : base;
        double fp = 0.0;   // pencil-constant part of the derivative factor
        if constexpr (DER) fp = kap.x * signed_mode(kx, kap.Nx) + kap.y * signed_mode(ky, Ny);
        // every lane is past the previous group's reads of the staged rows (the __syncwarp()s of its second pass)
        if (lane == 0) {
            mbar_arrive_expect_tx(gbar, G * Z::ROW * 8);
#pragma unroll
            for (int gg = 0; gg < G; ++gg) {
                int kx2, ky2;
                locate(grp * G + gg, kx2, ky2);
                const int qy2 = ky2 <= Ny ? ky2 : ny2 - ky2;
                bulk_load(gall + (warp * G + gg) * Z::ROW, Gk + ((long)kx2 * (Ny + 1) + qy2) * Z::ROW, Z::ROW * 8, gbar);
            }
        }
        double vr[R], vi[R];
#pragma unroll
        for (int i = 0; i < H; ++i) {   // the non-zero half of the padded pencil, and the first radix-2 level of the
            const double2 v = base[t + T * i];   // forward pass: (x_i, 0) -> (x_i, x_i)
            vr[i] = v.x; vi[i] = v.y;
            vr[i + H] = v.x; vi[i + H] = v.y;
        }
        if (grp + nwarps < (int)ngroups) {   // L2 prefetch of this lane group's next pencil: M * 16 / 128 lines
            int kx2, ky2;
            locate((grp + nwarps) * G + g, kx2, ky2);
            const double2* nb = B2 + ((long)kx2 * ny2 + ky2) * M;
#pragma unroll
            for (int e = 0; e < M / 8; e += T) asm volatile("prefetch.global.L2 [%0];" ::"l"(nb + (e + t) * 8));
        }
#pragma unroll 1
        for (int pass = 0; pass < 2; ++pass) {
            fft2_padded_pass<Cfg>(vr, vi, t, buf, cc, tn, pass);
            if (pass == 0) {   // Y = conj(Ghat X)
                mbar_wait(gbar, gpar);
                gpar ^= 1;
                const double fz0 = fp + kap.z * (double)t;   // DER only
                double kzv = kap.z;
                // opaque to the compiler: otherwise the 32 products kap.z * offset are formed once per kernel, spilled to
                // local memory and re-read for every pencil (35 doubles of spills)
                if constexpr (DER) asm volatile("" : "+d"(kzv));
#pragma unroll
                for (int i = 0; i < R; ++i) {
                    const double gk = i < H ? gA[T * i] : gB[-T * i];
                    if constexpr (DER) {
                        // signed mode of kz = t + T i: kz below M, kz - M2 above, zero at the Nyquist index kz = M
                        // (t = 0, i = R/2); the factor -i itself is applied to the final result (F^-1 is linear)
                        // (fz0 = fp + kap.z t, so at t = 0 the Nyquist factor fp is fz0 itself)
                        const double off = (double)(i < H ? T * i : T * i - M2);
                        const double cf = gk * ((i == H && t == 0) ? fz0 : fma(kzv, off, fz0));
                        vr[i] *= cf; vi[i] *= -cf;
                    } else {
                        vr[i] *= gk; vi[i] *= -gk;
                    }
                }
            }
        }
        // v = FFT(conj(Ghat X)) = conj(y): the kept half
#pragma unroll
        for (int i = 0; i < H; ++i)
            obase[t + T * i] = DER ? make_double2(-vi[i], -vr[i]) : make_double2(vr[i], -vi[i]);   // DER: -i y
    }
}

// =============================== K3 for Nz = 3 * 2^k (24 .. 384) and 5 * 2^k (40 .. 160): conv_z_pf, prime-factor warp kernel
// The zero-padded pencil of M2 = 2 Nz = B P points (B = 3 or 5, P = 16 .. 256) by the Good-Thomas map: with n = (P n1 + B n2)
// mod M2 on the input side and k = k1 (mod B), k = k2 (mod P) (CRT) on the output side,
//     X[k] = sum_n1 w_B^(n1 k1) sum_n2 w_P^(n2 k2) x[n]
// -- B P-point transforms (the warp-level two-stage transform of fft_warp.cuh, lane-constant twiddles, exchange
// private to the lane group) and a radix-B butterfly across them in registers, NO twiddles in between.  The DFT
// matrix is symmetric, so the same code also maps a CRT-ordered input to an (P n1 + B n2)-ordered output: the forward
// pass leaves the spectrum in CRT order (the spectrum rows are stored in that order, k_layout_spectrum_pfa), the
// inverse pass (IFFT(Y) = conj(FFT(conj Y)), the same copy of the code) returns to the order the pencil was loaded in.
// Against the CTA-level engine (k_conv_z_g2): no twiddle table, no CTA barriers, 8 free-running warps.
template <int B, int P>
struct ConvZPF {
    using Cfg = Fft2Cfg<P>;
    static constexpr int M2 = B * P, M = M2 / 2;           // M = Nz
    static constexpr int T = Cfg::T, R = Cfg::R;
    static constexpr int G = 32 / T;                       // pencils per warp
    static constexpr int WARPS = 8;
    static constexpr int ROW = M2;                         // doubles per spectrum row (CRT order, all M2 entries)
    static constexpr int NC = LaneTw<Cfg::R2>::NC;
    static constexpr int C1 = P * mod_inverse(P % B, B);   // k = (C1 k1 + C2 k2) mod M2:  P * (P^-1 mod B)
    static constexpr int C2 = B * mod_inverse(B % P, P);   //                              B * (B^-1 mod P)
    static_assert((B == 3 || B == 5) && C2 % P == 1 && C1 % B == 1, "CRT constants");
    // [exchange: WARPS*G*BUF double2][rows: WARPS*G*ROW doubles][mbarriers: WARPS]
    static constexpr size_t smem_bytes() {
        return sizeof(double2) * (size_t)(WARPS * G * Cfg::BUF) + sizeof(double) * (size_t)(WARPS * G * ROW) + 8 * WARPS;
    }
};

template <int B, int P, bool DER = false>
__global__ void __launch_bounds__(ConvZPF<B, P>::WARPS * 32, 1)
k_conv_z_pf(double2* __restrict__ B2, const double* __restrict__ Gk, const double* __restrict__ lane_g, int Ny,
            long ngroups, double2* __restrict__ out, const DerK kap) {
    using Z = ConvZPF<B, P>;
    using Cfg = typename Z::Cfg;
    constexpr int M = Z::M, M2 = Z::M2, R = Z::R, T = Z::T, G = Z::G, WARPS = Z::WARPS, NC = Z::NC, NB2 = Cfg::NB2;
    extern __shared__ double2 smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane / T, t = lane % T;
    double2* buf = smem + (warp * G + g) * Cfg::BUF;
    double* gall = reinterpret_cast<double*>(smem + WARPS * G * Cfg::BUF);
    const double* gst = gall + (warp * G + g) * Z::ROW;
    uint64_t* gbar = reinterpret_cast<uint64_t*>(gall + WARPS * G * Z::ROW) + warp;
    if (lane == 0) { mbar_init(gbar, 1); mbar_fence_init(); }
    __syncwarp();
    uint32_t gpar = 0;
    double cc[NB2][NC], tn[NB2][NC];
#pragma unroll
    for (int m = 0; m < NB2; ++m)
#pragma unroll
        for (int i = 0; i < NC; ++i) {
            cc[m][i] = lane_g[(t + T * m) * 2 * NC + i];
            tn[m][i] = lane_g[(t + T * m) * 2 * NC + NC + i];
        }
    const int nwarps = gridDim.x * WARPS;
    const int ny2 = 2 * Ny;
    auto locate = [&](int s_, int& kx_, int& ky_) {
        kx_ = s_ / ny2;
        const int r_ = s_ - kx_ * ny2;
        ky_ = (r_ & 1) ? ny2 - ((r_ + 1) >> 1) : (r_ >> 1);
    };
    for (int grp = blockIdx.x * WARPS + warp; grp < (int)ngroups; grp += nwarps) {
        int kx, ky;
        locate(grp * G + g, kx, ky);
        const double2* base = B2 + ((long)kx * ny2 + ky) * M;
        double2* obase = (DER ? out : B2) + ((long)kx * ny2 + ky) * M;
        double fp = 0.0;
        if constexpr (DER) fp = kap.x * signed_mode(kx, kap.Nx) + kap.y * signed_mode(ky, Ny);
        if (lane == 0) {   // every lane is past the previous group's reads of the staged rows
            mbar_arrive_expect_tx(gbar, G * Z::ROW * 8);
#pragma unroll
            for (int gg = 0; gg < G; ++gg) {
                int kx2, ky2;
                locate(grp * G + gg, kx2, ky2);
                const int qy2 = ky2 <= Ny ? ky2 : ny2 - ky2;
                bulk_load(gall + (warp * G + gg) * Z::ROW, Gk + ((long)kx2 * (Ny + 1) + qy2) * Z::ROW, Z::ROW * 8, gbar);
            }
        }
        // slot (n1, i) <-> n = (P n1 + B (t + T i)) mod M2; the padded half (n >= M) is zero
        double vr[B][R], vi[B][R];
#pragma unroll
        for (int n1 = 0; n1 < B; ++n1)
#pragma unroll
            for (int i = 0; i < R; ++i) {
                int n = P * n1 + B * (t + T * i);
                n -= n >= M2 ? M2 : 0;
                const double2 v = n < M ? base[n] : make_double2(0.0, 0.0);
                vr[n1][i] = v.x; vi[n1][i] = v.y;
            }
#pragma unroll 1
        for (int pass = 0; pass < 2; ++pass) {
#pragma unroll
            for (int n1 = 0; n1 < B; ++n1) fft2_forward_lc<Cfg>(vr[n1], vi[n1], t, buf, cc, tn);
#pragma unroll
            for (int i = 0; i < R; ++i) {   // radix B across the B sub-transforms (register stride R)
                double ar[B], ai[B];
#pragma unroll
                for (int n1 = 0; n1 < B; ++n1) { ar[n1] = vr[n1][i]; ai[n1] = vi[n1][i]; }
                if constexpr (B == 3) dft3<1>(ar, ai); else dft5<1>(ar, ai);
#pragma unroll
                for (int n1 = 0; n1 < B; ++n1) { vr[n1][i] = ar[n1]; vi[n1][i] = ai[n1]; }
            }
            if (pass == 0) {   // slot (k1, i) now holds X[k], k = k1 (mod B), k = t + T i (mod P); Y = conj(Ghat X)
                mbar_wait(gbar, gpar);
                gpar ^= 1;
#pragma unroll
                for (int k1 = 0; k1 < B; ++k1)
#pragma unroll
                    for (int i = 0; i < R; ++i) {
                        double gk = gst[k1 * P + t + T * i];
                        if constexpr (DER) {
                            const int k = (Z::C1 * k1 + Z::C2 * (t + T * i)) % M2;
                            gk *= fp + kap.z * signed_mode(k, M);
                        }
                        vr[k1][i] *= gk; vi[k1][i] *= -gk;
                    }
            }
        }
        // v = FFT(conj(Ghat X)) = conj(y), back in the order of the load; the kept half
#pragma unroll
        for (int n1 = 0; n1 < B; ++n1)
#pragma unroll
            for (int i = 0; i < R; ++i) {
                int n = P * n1 + B * (t + T * i);
                n -= n >= M2 ? M2 : 0;
                if (n < M) obase[n] = DER ? make_double2(-vi[n1][i], -vr[n1][i]) : make_double2(vr[n1][i], -vi[n1][i]);
            }
    }
}

// ====================================================================== K3 (v3, Nz = 512): conv_z_s
// The pair scheme of k_conv_z_p with the 32-lane transform of fft_warp.cuh (fft512s_forward): a warp holds ONE
// pencil branch with 16 points per lane, so the kernel needs half the registers (<= 128) and an SM runs 16 warps
// (8 pairs) instead of 8: with four warps per scheduler the fp64 phases of some warps overlap the shared-memory
// phases of the others (k_conv_z_p at 254 registers: fp64 pipe 59 %, 2 warps per scheduler).  Everything else as
// in k_conv_z_p: one copy of the transform run twice (IFFT(Y) = conj(FFT(conj(Y)))), octant spectrum rows staged by
// bulk async copies, the visiting order that lets two pencils share a row in L2, hand-over of v_o through the odd
// warp's exchange buffer under a pair barrier.
struct ConvZS {
    using F = Fft512S;
    static constexpr int M = 512, T = 32, R = 16;
    static constexpr int PAIRS = 8, WARPS = 2 * PAIRS;
    static constexpr int ROW = M + 2;
    // [wp: M double2][exchange: WARPS*BUF double2][G rows: PAIRS*ROW doubles][mbarriers: PAIRS]
    static constexpr size_t smem_bytes() {
        return sizeof(double2) * (size_t)(M + WARPS * F::BUF) + sizeof(double) * (size_t)(PAIRS * ROW) + 8 * PAIRS;
    }
};

template <bool DER = false>
__global__ void __launch_bounds__(ConvZS::WARPS * 32, 1)
k_conv_z_s(double2* __restrict__ B2, const double* __restrict__ Gk, const double* __restrict__ lane_g,
           const double2* __restrict__ wp_g, int Ny, long nsteps, double2* __restrict__ out, const DerK kap) {
    using Z = ConvZS;
    using F = Fft512S;
    constexpr int M = Z::M, R = Z::R, T = Z::T, PAIRS = Z::PAIRS, WARPS = Z::WARPS, NC = F::NC;
    extern __shared__ double2 smem[];
    double2* wp = smem;          // M: w_2M^n, n < M
    for (int n = threadIdx.x; n < M; n += blockDim.x) wp[n] = wp_g[n];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, q = warp >> 1, b = warp & 1;
    const int t = lane;
    double2* buf = smem + M + warp * F::BUF;
    double2* pbuf = smem + M + (warp ^ 1) * F::BUF;          // the partner's buffer
    double* gall = reinterpret_cast<double*>(smem + M + WARPS * F::BUF);
    double* gst = gall + q * Z::ROW;
    uint64_t* gbar = reinterpret_cast<uint64_t*>(gall + PAIRS * Z::ROW) + q;
    if (b == 0 && lane == 0) { mbar_init(gbar, 1); mbar_fence_init(); }
    __syncthreads();
    uint32_t gpar = 0;
    double cc[NC], tn[NC], xc[8], xt[8];
#pragma unroll
    for (int i = 0; i < NC; ++i) {
        cc[i] = lane_g[t * 2 * NC + i];
        tn[i] = lane_g[t * 2 * NC + NC + i];
    }
#pragma unroll
    for (int m = 0; m < 8; ++m) {
        xc[m] = lane_g[32 * 2 * NC + (lane >> 4) * 16 + m];
        xt[m] = lane_g[32 * 2 * NC + (lane >> 4) * 16 + 8 + m];
    }
    const int npairs = gridDim.x * PAIRS;
    const int ny2 = 2 * Ny;
    auto locate = [&](int s_, int& kx_, int& ky_) {   // position in the visiting order -> (kx, ky)
        kx_ = s_ / ny2;
        const int r_ = s_ - kx_ * ny2;
        ky_ = (r_ & 1) ? ny2 - ((r_ + 1) >> 1) : (r_ >> 1);
    };
    for (int step = blockIdx.x * PAIRS + q; step < (int)nsteps; step += npairs) {
        int kx, ky;
        locate(step, kx, ky);
        const int qy = ky <= Ny ? ky : ny2 - ky;
        double2* base = B2 + ((long)kx * ny2 + ky) * M;
        double2* obase = DER ? out + ((long)kx * ny2 + ky) * M : base;
        double fp = 0.0;
        if constexpr (DER) fp = kap.x * signed_mode(kx, kap.Nx) + kap.y * signed_mode(ky, Ny);
        // both warps are past the previous step's reads of the staged row (the pair barrier ending the combine)
        if (b == 0 && lane == 0) {
            mbar_arrive_expect_tx(gbar, Z::ROW * 8);
            bulk_load(gst, Gk + ((long)kx * (Ny + 1) + qy) * Z::ROW, Z::ROW * 8, gbar);
        }
        double vr[R], vi[R];
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const double2 v = base[t + T * i];
            vr[i] = v.x; vi[i] = v.y;
        }
        if (step + npairs < (int)nsteps) {   // L2 prefetch of the pair's next pencil, half of the lines from each warp
            int kx2, ky2;
            locate(step + npairs, kx2, ky2);
            const double2* nb = B2 + ((long)kx2 * ny2 + ky2) * M;
            asm volatile("prefetch.global.L2 [%0];" ::"l"(nb + (b * 32 + lane) * 8));   // 64 lines of 128 bytes
        }
        if (b) {
#pragma unroll
            for (int i = 0; i < R; ++i) cmul(vr[i], vi[i], wp[t + T * i]);
        }
#pragma unroll 1
        for (int pass = 0; pass < 2; ++pass) {
            fft512s_forward(vr, vi, lane, buf, cc, tn, xc, xt);
            if (pass == 0) {
                mbar_wait(gbar, gpar);
                gpar ^= 1;
                const double* gsrc = gst + (b ? M / 2 + 1 : 0);
                const double* gA = gsrc + t;
                const double* gB = gsrc + (M - b - t);
                const double fz0 = fp + kap.z * (double)(2 * t + b);   // DER only
                const bool nyq = (2 * t + b) == 0;                      // register R/2 of this lane is kz = M
#pragma unroll
                for (int i = 0; i < R; ++i) {
                    const double gk = i < R / 2 ? gA[T * i] : gB[-T * i];   // row index min(j, M-b-j), j = t + T i
                    if constexpr (DER) {
                        double cf = gk * fma(kap.z, (double)(i < R / 2 ? 2 * T * i : 2 * T * i - 2 * M), fz0);
                        if (i == R / 2) cf = nyq ? gk * fp : cf;
                        vr[i] *= cf; vi[i] *= -cf;
                    } else {
                        vr[i] *= gk; vi[i] *= -gk;
                    }
                }
            }
        }
        // v = FFT(conj(Ghat X)) on each branch; y[n] = conj(v_e[n] + w^n v_o[n]), formed by the even warp
        if (b) {
            __syncwarp();   // this warp's exchange reads are complete: buf becomes the outbox
#pragma unroll
            for (int i = 0; i < R; ++i) buf[t + T * i] = make_double2(vr[i], vi[i]);
        }
        bar_sync(1 + q, 64);
        if (!b) {
#pragma unroll
            for (int i = 0; i < R; ++i) {
                const double2 pv = pbuf[t + T * i];   // v_o[n], n = t + T i
                const double2 w = wp[t + T * i];
                const double zr = fma(-w.y, pv.y, fma(w.x, pv.x, vr[i]));
                const double zi = fma(w.y, pv.x, fma(w.x, pv.y, vi[i]));
                obase[t + T * i] = DER ? make_double2(-zi, -zr) : make_double2(zr, -zi);   // DER: -i y
            }
        }
        bar_sync(1 + q, 64);   // the even warp has read the outbox (and both are done with the staged row)
    }
}

// ================================================================================ K1 (v2): fwd_x_r2c_t
// Tile kernel for the real-to-complex pass along x (M = Nx/2 complex points z[n] = rho[2n] + i rho[2n+1]).
// Tile = all Nx rows of kC = 16 adjacent columns of the flattened (y, z) plane (one 128-byte line of
// doubles per row), delivered by TMA through a 2-D tensor map over rho.  Group 0 computes Z[2j], group 1
// Z[2j+1] (input times w_N^n); the untangling partner Z[N-k] has the parity of k, so it is found inside
// the group: the group's exchange buffer is reused to look it up.  The twiddles w_2N^k and w_N^n factor
// into a per-lane constant times a compile-time 32nd root of unity (k = (2t+g) + 2T i, n = t + T i,
// N/T = 32 or 16), so no twiddle table is read.
constexpr int kC = 16;
template <int M>
struct TileX {
    using Cfg = Fft2Cfg<M>;
    static constexpr int T = Cfg::T, R = Cfg::R;
    static constexpr int ROOT = 2 * M / T;        // N/T: the compile-time roots are w_ROOT^i
    static_assert(64 % ROOT == 0, "tile x kernels need N/T to divide 64");
    static constexpr int WS = ROOT <= 32 ? 32 / ROOT : 1;   // w_ROOT^i = w_32^(WS i), or w_64^i when ROOT = 64
    static constexpr int KC = (M >= 512) ? 8 : kC;   // columns per tile (Nx = 1024: 8, registers and shared memory)
    static constexpr int GT = KC * T, THREADS = 2 * GT;
    static constexpr int NC = LaneTw<Cfg::R2>::NC;
    static constexpr int MINB = (M >= 256) ? 1 : 2;
    // [mbarriers: 128 B][X: 2M rows x kC doubles = M*kC double2][E: 2 groups x M*kC double2]
    static constexpr size_t smem_bytes() { return 128 + sizeof(double2) * (size_t)(3 * M * KC); }
};

// x * w_32^i (compile-time i)
template <int i>
__device__ __forceinline__ void cmul_w32(double& xr, double& xi) {
    if constexpr ((i & 31) == 0) {
    } else if constexpr ((i & 31) == 8) {   // -i
        const double a = xi; xi = -xr; xr = a;
    } else {
        const double c = cos32(i), sn = sin32(i);
        const double a = fma(xi, sn, xr * c);
        xi = fma(-xr, sn, xi * c);
        xr = a;
    }
}

// x * w_64^i (compile-time i)
template <int i>
__device__ __forceinline__ void cmul_w64(double& xr, double& xi) {
    if constexpr ((i & 63) == 0) {
    } else if constexpr ((i & 63) == 16) {   // -i
        const double a = xi; xi = -xr; xr = a;
    } else {
        const double c = cos64(i), sn = sin64(i);
        const double a = fma(xi, sn, xr * c);
        xi = fma(-xr, sn, xi * c);
        xr = a;
    }
}
template <int i>
__device__ __forceinline__ void cmul_w64c(double& xr, double& xi) {   // x * conj(w_64^i)
    if constexpr ((i & 63) == 0) {
    } else if constexpr ((i & 63) == 16) {   // +i
        const double a = -xi; xi = xr; xr = a;
    } else {
        const double c = cos64(i), sn = sin64(i);
        const double a = fma(-xi, sn, xr * c);
        xi = fma(xr, sn, xi * c);
        xr = a;
    }
}

template <int M, int I = 0>
struct UntangleFwd {   // unrolled over the register index with compile-time roots
    template <class F>
    __device__ __forceinline__ static void run(F&& f) {
        if constexpr (I < Fft2Cfg<M>::R) {
            f(std::integral_constant<int, I>{});
            UntangleFwd<M, I + 1>::run(f);
        }
    }
};

template <int M>
__global__ void __launch_bounds__(TileX<M>::THREADS, TileX<M>::MINB)
k_fwd_x_t(const __grid_constant__ CUtensorMap tmRho, double2* __restrict__ B1, const double* __restrict__ lane_g,
          const double2* __restrict__ Wg, long plane, long ntiles) {
    using X_ = TileX<M>;
    using Cfg = typename X_::Cfg;
    constexpr int R = X_::R, T = X_::T, GT = X_::GT, NC = X_::NC, NB2 = Cfg::NB2, N = 2 * M, KC = X_::KC;
    constexpr int BOXR = N < 256 ? N : 256;
    extern __shared__ __align__(128) unsigned char smraw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smraw);
    double* Xd = reinterpret_cast<double*>(smraw + 128);
    double2* E = reinterpret_cast<double2*>(smraw + 128) + M * KC;
    const int tid = threadIdx.x;
    const int grp = tid / GT, gt = tid % GT, c = gt % KC, t = gt / KC;
    double cc[NB2][NC], tn[NB2][NC];
#pragma unroll
    for (int m = 0; m < NB2; ++m)
#pragma unroll
        for (int i = 0; i < NC; ++i) {
            cc[m][i] = lane_g[(t + T * m) * 2 * NC + i];
            tn[m][i] = lane_g[(t + T * m) * 2 * NC + NC + i];
        }
    const double2 lam_n = Wg[2 * t];          // w_N^t     (Wg[m] = exp(-2 pi i m / 2N))
    const double2 lam_k = Wg[2 * t + grp];    // w_2N^(2t+g)
    // full: the tile has landed in X; empty (full + 1): every thread holds its part of it.  The two groups are NOT
    // synchronised with one another: group 1 (which has the pre-twiddle on top) falls behind until it reads a tile just
    // before group 0 wants the next one, and from then on the shared-memory phases of one group run under the fp64
    // phases of the other (a CTA-wide barrier here kept all 16 warps in the same phase)
    uint64_t* empty = full + 1;
    if (tid == 0) { mbar_init(full, 1); mbar_init(empty, X_::THREADS); mbar_fence_init(); }
    __syncthreads();
    auto issue = [&](long tile) {
        mbar_arrive_expect_tx(full, (uint32_t)(N * KC * sizeof(double)));
#pragma unroll
        for (int r0 = 0; r0 < N; r0 += BOXR) tma_load_2d(Xd + r0 * KC, &tmRho, full, (int)(tile * KC), r0);
    };
    long tile = blockIdx.x;
    if (tid == 0 && tile < ntiles) issue(tile);
    uint32_t parity = 0;
    double2* Ec = E + grp * (M * KC) + c;
    for (; tile < ntiles; tile += gridDim.x) {
        double vr[R], vi[R];
        mbar_wait(full, parity);
        parity ^= 1;
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const int n = t + T * i;
            vr[i] = Xd[(2 * n) * KC + c];
            vi[i] = Xd[(2 * n + 1) * KC + c];
        }
        mbar_arrive(empty);
        if (tid == GT && tile + gridDim.x < ntiles) {   // first thread of group 1: X may be refilled once both groups hold the tile
            mbar_wait(empty, parity ^ 1);
            issue(tile + gridDim.x);
        }
        if (grp) {   // z[n] w_N^n,  w_N^n = w_N^t w_32^i
            UntangleFwd<M>::run([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                cmul(vr[i], vi[i], lam_n);
                if constexpr (X_::ROOT <= 32) cmul_w32<i * X_::WS>(vr[i], vi[i]); else cmul_w64<i>(vr[i], vi[i]);
            });
        }
        fft2_forward_tile<Cfg, KC>(vr, vi, t, Ec, 1 + grp, cc, tn);
        // untangle: X'[k] = (A + B) - i w_2N^k (A - B), A = Z[k], B = conj(Z[N-k]), k = 2j + g, j = t + T i
        bar_sync(1 + grp, GT);   // exchange buffer read back by the whole group
#pragma unroll
        for (int i = 0; i < R; ++i) Ec[(t + T * i) * KC] = make_double2(vr[i], vi[i]);
        bar_sync(1 + grp, GT);
        double2* out = B1 + tile * KC + c;
        UntangleFwd<M>::run([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            const int j = t + T * i;
            const int jp = grp ? M - 1 - j : (M - j) & (M - 1);
            const double2 bq = Ec[jp * KC];
            const double ar = vr[i], ai = vi[i], br = bq.x, bi = -bq.y;
            const double sr = ar + br, si = ai + bi;
            double dr = ar - br, di = ai - bi;
            cmul(dr, di, lam_k);
            if constexpr (X_::ROOT <= 32) cmul_w32<i * X_::WS>(dr, di); else cmul_w64<i>(dr, di);
            const long k = 2 * j + grp;
            out[k * plane] = make_double2(sr + di, si - dr);
            if (i == 0 && grp == 0 && t == 0) out[(long)N * plane] = make_double2(2.0 * (ar - ai), 0.0);
        });
    }
}

// ================================================================================ K5 (v2): inv_x_c2r_t
// Tile kernel for the complex-to-real pass along x, mirror image of k_fwd_x_t.  Group g rebuilds
// Z[2j+g] = (A + B) + i conj(w_2N^k)(A - B), A = X[k], B = conj(X[N-k]) (N - k has the parity of k, so each
// group needs the rows of its own parity only: 3-D tensor map [j][parity][2 plane doubles]; row N, needed
// by k = 0, comes by a separate bulk copy), inverse-transforms it in place in its buffer, and
// y[n] = y_e[n] + conj(w_N^n) y_o[n] gives phi[2n] = Re y[n], phi[2n+1] = Im y[n]: the restriction of
// PAPER.md:82 is simply that rows n >= Nx/2 are never formed.
template <int i>
__device__ __forceinline__ void cmul_w32c(double& xr, double& xi) {   // x * conj(w_32^i)
    if constexpr ((i & 31) == 0) {
    } else if constexpr ((i & 31) == 8) {   // +i
        const double a = -xi; xi = xr; xr = a;
    } else {
        const double c = cos32(i), sn = sin32(i);
        const double a = fma(-xi, sn, xr * c);
        xi = fma(xr, sn, xi * c);
        xr = a;
    }
}

template <int M>
struct TileXI {
    using Cfg = Fft2Cfg<M>;
    static constexpr int T = Cfg::T, R = Cfg::R;
    static constexpr int ROOT = 2 * M / T;
    static_assert(64 % ROOT == 0, "tile x kernels need N/T to divide 64");
    static constexpr int WS = ROOT <= 32 ? 32 / ROOT : 1;   // w_ROOT^i = w_32^(WS i), or w_64^i when ROOT = 64
    static constexpr int KC = (M >= 512) ? 8 : kC;
    static constexpr int GT = KC * T, THREADS = 2 * GT;
    static constexpr int NC = LaneTw<Cfg::R2>::NC;
    static constexpr int MINB = (M >= 256) ? 1 : 2;
    static constexpr int BOXR = M < 256 ? M : 256;
    // [mbarriers: 128 B][row N: KC double2][X: 2 groups x M*KC][C: 2 groups x (M/2)*KC]
    static constexpr size_t smem_bytes() { return 128 + sizeof(double2) * (size_t)(KC + 3 * M * KC); }
};

// DER: X[k] is multiplied by -i kder k first (zero at the Nyquist index k = Nx): E_x of the field output
template <int M, bool DER = false>
__global__ void __launch_bounds__(TileXI<M>::THREADS, TileXI<M>::MINB)
k_inv_x_t(const __grid_constant__ CUtensorMap tmB1, const double2* __restrict__ B1, double* __restrict__ phi,
          const double* __restrict__ lane_g, const double2* __restrict__ Wg, long plane, long ntiles, const double kder) {
    using X_ = TileXI<M>;
    using Cfg = typename X_::Cfg;
    constexpr int R = X_::R, T = X_::T, GT = X_::GT, NC = X_::NC, NB2 = Cfg::NB2, N = 2 * M, H = R / 2, KC = X_::KC;
    extern __shared__ __align__(128) unsigned char smraw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smraw);
    double2* XN = reinterpret_cast<double2*>(smraw + 128);
    double2* X = XN + KC;
    double2* C = X + 2 * M * KC;
    const int tid = threadIdx.x;
    const int grp = tid / GT, gt = tid % GT, c = gt % KC, t = gt / KC;
    double cc[NB2][NC], tn[NB2][NC];
#pragma unroll
    for (int m = 0; m < NB2; ++m)
#pragma unroll
        for (int i = 0; i < NC; ++i) {
            cc[m][i] = lane_g[(t + T * m) * 2 * NC + i];
            tn[m][i] = lane_g[(t + T * m) * 2 * NC + NC + i];
        }
    const double2 lam_n = Wg[2 * t];          // w_N^t
    const double2 lam_k = Wg[2 * t + grp];    // w_2N^(2t+g)
    const double kd0 = kder * (double)(2 * t + grp);   // DER only
    if (tid == 0) { mbar_init(&full[0], 1); mbar_init(&full[1], 1); mbar_fence_init(); }
    __syncthreads();
    double2* Xg = X + grp * (M * KC);
    auto issue = [&](long tile) {   // one thread of the group
        const uint32_t bytes = (uint32_t)(M * KC * sizeof(double2)) + (grp == 0 ? (uint32_t)(KC * sizeof(double2)) : 0u);
        mbar_arrive_expect_tx(&full[grp], bytes);
#pragma unroll
        for (int r0 = 0; r0 < M; r0 += X_::BOXR) tma_load_3d(Xg + r0 * KC, &tmB1, &full[grp], (int)(tile * KC * 2), grp, r0);
        if (grp == 0) bulk_load(XN, B1 + (long)N * plane + tile * KC, KC * sizeof(double2), &full[0]);
    };
    auto prefetch = [&](long tile) {
#pragma unroll
        for (int r0 = 0; r0 < M; r0 += X_::BOXR) tma_prefetch_3d(&tmB1, (int)(tile * KC * 2), grp, r0);
    };
    long tile = blockIdx.x;
    if (gt == 0 && tile < ntiles) issue(tile);
    uint32_t parity = 0;
    double2* Ec = Xg + c;
    double2* Cmine = C + grp * (M / 2 * KC) + c;
    double2* Ctheirs = C + (grp ^ 1) * (M / 2 * KC) + c;
    for (; tile < ntiles; tile += gridDim.x) {
        const bool more = tile + gridDim.x < ntiles;
        if (gt == 0 && more) prefetch(tile + gridDim.x);
        double zr[R], zi[R];
        mbar_wait(&full[grp], parity);
        parity ^= 1;
        double kdv = kder;   // opaque: keeps the 2 R mode factors from being formed once per kernel and spilled (DER only)
        if constexpr (DER) asm volatile("" : "+d"(kdv));
        UntangleFwd<M>::run([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            const int j = t + T * i;
            double2 a = Ec[j * KC];
            double2 bq;
            if (grp) bq = Ec[(M - 1 - j) * KC];
            else bq = (j == 0) ? XN[c] : Ec[(M - j) * KC];
            if constexpr (DER) {   // k = (2t + grp) + 2T i: a lane constant plus a compile-time multiple
                const double ck = fma(kdv * (double)(2 * T), (double)i, kd0);
                mul_minus_i(a.x, a.y, ck);
                mul_minus_i(bq.x, bq.y, (i == 0 && kd0 == 0.0) ? 0.0 : kdv * (double)N - ck);   // N - k; row N is the Nyquist row
            }
            const double br = bq.x, bi = -bq.y;
            const double sr = a.x + br, si = a.y + bi;
            double dr = a.x - br, di = a.y - bi;
            cmul_conj(dr, di, lam_k);
            if constexpr (X_::ROOT <= 32) cmul_w32c<i * X_::WS>(dr, di); else cmul_w64c<i>(dr, di);
            zr[i] = sr - di; zi[i] = si + dr;     // Z = (A + B) + i d
        });
        fft2_forward_tile<Cfg, KC>(zi, zr, t, Ec, 1 + grp, cc, tn);   // inverse: roles of re and im swapped
        bar_sync(1 + grp, GT);   // exchange read back: X_g is free
        if (gt == 0 && more) { fence_proxy_async(); issue(tile + gridDim.x); }
        if (grp) {   // y_o[n] conj(w_N^n), n = t + T i
            UntangleFwd<M>::run([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                cmul_conj(zr[i], zi[i], lam_n);
                if constexpr (X_::ROOT <= 32) cmul_w32c<i * X_::WS>(zr[i], zi[i]); else cmul_w64c<i>(zr[i], zi[i]);
            });
        }
        __syncthreads();         // C of the previous tile has been consumed
#pragma unroll
        for (int i = 0; i < H; ++i) {
            Cmine[(t + T * i) * KC] = make_double2(grp ? zr[i] : zr[i + H], grp ? zi[i] : zi[i + H]);
        }
        __syncthreads();
        double* out = phi + tile * KC + c;
#pragma unroll
        for (int i = 0; i < H; ++i) {
            const double2 pv = Ctheirs[(t + T * i) * KC];
            const int o = grp ? i + H : i;
            const long n = t + T * o;
            out[(2 * n) * plane] = (grp ? zr[i + H] : zr[i]) + pv.x;
            out[(2 * n + 1) * plane] = (grp ? zi[i + H] : zi[i]) + pv.y;
        }
    }
}

// ================================================================================== K1: fwd_x_r2c
// M = Nx/2.  Tile = (y, z-bundle of kW columns); rows are x.  LTAB = 2Nx = 4M.
template <int M>
__global__ void __launch_bounds__(TileGroups<FftCfg<M>>::G* kW* FftCfg<M>::T)
k_fwd_x_r2c(const double* __restrict__ rho, double2* __restrict__ B1, const double2* __restrict__ Wg,
            int Ny, int Nz, long ntiles) {
    using Cfg = FftCfg<M>;
    constexpr int R = Cfg::R, T = Cfg::T, G = TileGroups<Cfg>::G, LTAB = 4 * M, N = 2 * M;
    extern __shared__ double2 smem[];
    double2* Ws = smem;                      // LTAB
    double2* xb = Ws + LTAB;                 // G * M * kW   exchange
    double2* zs = xb + G * M * kW;           // G * N * kW   Z[k] for the untangling
    load_table<LTAB>(Ws, Wg);
    const int tid = threadIdx.x;
    const int g = tid / (kW * T), lt = tid % (kW * T);
    const int c = lt % kW, t = lt / kW;
    double2* buf = xb + g * (M * kW) + c;
    double2* Z = zs + g * (N * kW) + c;
    const long tile = (long)blockIdx.x * G + g;
    const bool valid = tile < ntiles;
    const int nzb = Nz / kW;
    const long y = valid ? tile / nzb : 0;
    const int zb = valid ? (int)(tile % nzb) : 0;
    const long plane = (long)Ny * Nz;
    const double* in = rho + y * Nz + zb * kW + c;
    double2* out = B1 + y * Nz + zb * kW + c;

    double xr[R], xi[R], vr[R], vi[R];
#pragma unroll
    for (int i = 0; i < R; ++i) {
        const long n = t + T * i;
        xr[i] = valid ? in[(2 * n) * plane] : 0.0;
        xi[i] = valid ? in[(2 * n + 1) * plane] : 0.0;
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < R; ++i) { vr[i] = xr[i]; vi[i] = xi[i]; }
    fft_forward<Cfg, kW, LTAB>(vr, vi, t, buf, Ws);
#pragma unroll
    for (int i = 0; i < R; ++i) Z[(2 * (t + T * i)) * kW] = make_double2(vr[i], vi[i]);
    // odd: z[n] * w_N^n = W[2n] (table is exp(-2 pi i n/(2N)))
#pragma unroll
    for (int i = 0; i < R; ++i) cmul(xr[i], xi[i], Ws[2 * (t + T * i)]);
    fft_forward<Cfg, kW, LTAB>(xr, xi, t, buf, Ws);
#pragma unroll
    for (int i = 0; i < R; ++i) Z[(2 * (t + T * i) + 1) * kW] = make_double2(xr[i], xi[i]);
    __syncthreads();
    if (valid) {
#pragma unroll
        for (int i = 0; i < R; ++i) {
#pragma unroll
            for (int o = 0; o < 2; ++o) {
                const int k = 2 * (t + T * i) + o;
                const double2 a = Z[k * kW];
                const double2 bq = Z[(k == 0 ? 0 : N - k) * kW];
                const double br = bq.x, bi = -bq.y;            // B = conj(Z[N-k])
                const double sr = a.x + br, si = a.y + bi;     // A + B
                double dr = a.x - br, di = a.y - bi;           // A - B
                cmul(dr, di, Ws[k]);                           // w^k (A - B)
                // X' = (A+B) - i * d = (sr + di) + i (si - dr)
                out[(long)k * plane] = make_double2(sr + di, si - dr);
                if (k == 0) {
                    // k = N: A = Z[0], B = conj(Z[0]), w^N = -1  ->  X'[N] = 2 (Re Z0 - Im Z0)
                    out[(long)N * plane] = make_double2(2.0 * (a.x - a.y), 0.0);
                }
            }
        }
    }
}

// ================================================================================== K5: inv_x_c2r
template <int M, bool DER = false>
__global__ void __launch_bounds__(TileGroups<FftCfg<M>>::G* kW* FftCfg<M>::T)
k_inv_x_c2r(const double2* __restrict__ B1, double* __restrict__ phi, const double2* __restrict__ Wg,
            int Ny, int Nz, long ntiles, const double kder) {
    using Cfg = FftCfg<M>;
    constexpr int R = Cfg::R, T = Cfg::T, G = TileGroups<Cfg>::G, LTAB = 4 * M, N = 2 * M;
    extern __shared__ double2 smem[];
    double2* Ws = smem;
    double2* xb = Ws + LTAB;
    load_table<LTAB>(Ws, Wg);
    const int tid = threadIdx.x;
    const int g = tid / (kW * T), lt = tid % (kW * T);
    const int c = lt % kW, t = lt / kW;
    double2* buf = xb + g * (M * kW) + c;
    const long tile = (long)blockIdx.x * G + g;
    const bool valid = tile < ntiles;
    const int nzb = Nz / kW;
    const long y = valid ? tile / nzb : 0;
    const int zb = valid ? (int)(tile % nzb) : 0;
    const long plane = (long)Ny * Nz;
    const double2* in = B1 + y * Nz + zb * kW + c;
    double* out = phi + y * Nz + zb * kW + c;

    double er[R], ei[R], qr[R], qi[R];
    __syncthreads();  // table (needed while building Z)
#pragma unroll
    for (int i = 0; i < R; ++i) {
#pragma unroll
        for (int o = 0; o < 2; ++o) {
            const int k = 2 * (t + T * i) + o;
            double2 a = valid ? in[(long)k * plane] : make_double2(0.0, 0.0);
            double2 bq = valid ? in[(long)(N - k) * plane] : make_double2(0.0, 0.0);
            if constexpr (DER) {
                mul_minus_i(a.x, a.y, kder * (double)k);
                mul_minus_i(bq.x, bq.y, k == 0 ? 0.0 : kder * (double)(N - k));
            }
            const double br = bq.x, bi = -bq.y;
            const double sr = a.x + br, si = a.y + bi;
            double dr = a.x - br, di = a.y - bi;
            cmul_conj(dr, di, Ws[k]);                      // conj(w^k) (A - B)
            // Z = (A+B) + i d = (sr - di) + i (si + dr)
            if (o == 0) { er[i] = sr - di; ei[i] = si + dr; }
            else        { qr[i] = sr - di; qi[i] = si + dr; }
        }
    }
    fft_inverse<Cfg, kW, LTAB>(qr, qi, t, buf, Ws);
#pragma unroll
    for (int i = 0; i < R; ++i) cmul_conj(qr[i], qi[i], Ws[2 * (t + T * i)]);
    fft_inverse<Cfg, kW, LTAB>(er, ei, t, buf, Ws);
    if (valid) {
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const long n = t + T * i;
            out[(2 * n) * plane] = er[i] + qr[i];
            out[(2 * n + 1) * plane] = ei[i] + qi[i];
        }
    }
}

}  // namespace fsp

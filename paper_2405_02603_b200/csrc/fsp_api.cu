// fsp_api.cu -- the C ABI of include/fsp.h: plan management, Green precompute driver, and the
// five-kernel solve.  Host code only marshals sizes and launches; every step of the path runs in the
// kernels of solve_kernels.cuh / green_kernels.cuh.
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <new>
#include <atomic>
#include <vector>

#include <cuda.h>
#include <cuda_runtime.h>

#include "../../include/fsp.h"
#include "green_kernels.cuh"
#include "solve_kernels.cuh"
#include "shard.cuh"
#include "ubench.cuh"
#include "periodic_kernels.cuh"

using namespace fsp;

#define FSP_VERSION_NUM 200

struct fsp_plan {
    int Nx = 0, Ny = 0, Nz = 0;   // transform mesh: each a power of two (the caller's mesh when that is one)
    int Ux = 0, Uy = 0, Uz = 0;   // the caller's mesh; U_d <= N_d
    bool padded = false;          // U != N: rho is embedded in / phi cropped from the transform mesh (R19)
    double *rho_pad = nullptr, *phi_pad = nullptr;   // Nx*Ny*Nz each, only when padded
    double h[3] = {0, 0, 0};
    int algorithm = 0;
    cudaStream_t stream = nullptr;
    int device = 0;
    double g0 = 0.0, alpha = 1.1;
    int vg_m[3] = {4, 4, 4};  // oversampling factors used by the last VG precompute
    // plan-owned device memory
    double2* B1 = nullptr;  // (Nx+1) * Ny * Nz
    double2* B2 = nullptr;  // (Nx+1) * 2Ny * Nz
    double* Gk = nullptr;   // (Nx+1)(Ny+1)(Nz+2)   spectrum octant in K3's layout, scale folded in
    double* LTz = nullptr;  // lane-constant stage-2 twiddles of the z transform (fft_warp.cuh dft_lane)
    double* LTzs = nullptr; // Nz = 512: constants of the 32-lane transform (k_conv_z_s): stage 2 [32][16], shuffled level [2][16]
    double* LTzf = nullptr; // Nz = 256, 512: stage-2 constants of the padded transform of 2 Nz points (k_conv_z_f)
    int k3_variant = 0;     // FSP_PARAM_K3_VARIANT
    // shape of the workspace (sharded plans): a whole plan holds Nx + 1 kx planes and runs all five passes
    int stage = 0;          // 0: whole solve; 1: x passes only (K1, K5); 2: the y-z-y middle only (K2, K3, K4)
    int planes = 0;         // kx planes held by B1 (stage 2), B2 and Gk; Nx + 1 unless stage 2 of a sharded plan
    int kx0 = 0;            // global index of the first of them
    size_t b1_count = 0, b2_count = 0;   // complex elements allocated in B1, B2
    // warp-level DCT-I of the precompute: per transform length M, the lane-constant table and the roots exp(-2 pi i m / 2M)
    std::vector<int> dct_len;
    std::vector<double*> dct_lane;
    std::vector<double2*> dct_roots;
    bool gk_pfa = false;     // Gk rows hold all 2 Nz entries in CRT order (k_conv_z_pf, Nz = 96, 192, 384)
    bool gk_natural = false; // Gk rows in natural order (k_conv_z_f) instead of [E | O] (decided by the last precompute)
    double* LTy = nullptr;  // the same for the y transform (tile kernels)
    double* LTyf = nullptr; // Ny = 512: stage-2 constants of the padded 1024-point y transform (k_fwd_y_f)
    int k2_variant = 0;     // FSP_PARAM_K2_VARIANT
    bool periodic_fast_z = true;   // FSP_PARAM_PERIODIC_FAST_Z: periodic z (Nz = 2^k) by Nz-point transforms (k_conv_z_periodic)
    int periodic = 0;       // FSP_PARAM_PERIODIC: bit d set = direction d periodic (nearest-image kernel of period N_d h_d)
    bool tile_y = false;    // K2/K4 tile kernels (TMA-staged) are used
    double* LTx = nullptr;  // lane-constant twiddles of the x transform (length Nx/2)
    bool tile_x = false;    // K1 tile kernel is used
    CUtensorMap tmRho;      // rho as [x][Ny*Nz doubles], box = 16 columns x <=256 rows; re-encoded when rho moves
    const double* tmRho_ptr = nullptr;
    CUtensorMap tmB1x;      // B1 as [j][parity][2 Ny Nz doubles] (row = 2j + parity), box = 16 columns x 1 x <=256 (K5 input)
    CUtensorMap tmB1y;      // B1 as [kx][y][2 Nz doubles], box = 8 columns x <=256 rows (K2 input)
    CUtensorMap tmB2y;      // B2 as [kx][j][parity][2 Nz doubles], box = 8 columns x 1 parity x <=256 j (K4 input)
    double2* B3 = nullptr;  // second B2-sized buffer, allocated by the first fsp_solve_field (derivative spectra)
    CUtensorMap tmB3y;      // the same view of B3
    int chunk_planes = 0;   // > 0: K2-K3-K4 run chunk_planes kx-planes at a time (L2-resident B2)
    int sm_count = 148;
    double* T = nullptr;    // (Nx+1)(Ny+1)(Nz+1)   real-space table
    double* Goct = nullptr; // (Nx+1)(Ny+1)(Nz+1)   un-normalised spectrum octant
    double2 *Wx = nullptr, *Wy = nullptr, *Wz = nullptr;  // exp(-2 pi i n / 2N_d), n < 2N_d
    double *rho_stage = nullptr, *phi_stage = nullptr, *E_stage = nullptr;
    // fsp_solve_host_batch: second pair of staging buffers, copy streams, hand-off events (created on first use)
    double *rho_stage2 = nullptr, *phi_stage2 = nullptr;
    cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
    cudaEvent_t ev_h2d[2] = {nullptr, nullptr}, ev_solve[2] = {nullptr, nullptr}, ev_d2h[2] = {nullptr, nullptr};
    bool precomputed = false;
    size_t bytes = 0, peak_transient = 0;
    // profiling
    bool profiling = false;
    std::vector<cudaEvent_t> events;  // 6 per recorded solve
    size_t events_used = 0;
};

namespace {

int map_cuda(cudaError_t e) {
    if (e == cudaSuccess) return FSP_OK;
    if (e == cudaErrorMemoryAllocation) return FSP_ERR_OUT_OF_MEMORY;
    if (e == cudaErrorNoDevice || e == cudaErrorInsufficientDriver) return FSP_ERR_NO_DEVICE;
    return FSP_ERR_CUDA;
}

#define CU(call)                                     \
    do {                                             \
        cudaError_t e__ = (call);                    \
        if (e__ != cudaSuccess) {                    \
            (void)cudaGetLastError();                \
            return map_cuda(e__);                    \
        }                                            \
    } while (0)

template <class T>
int dev_alloc(T** p, size_t count, size_t* acc) {
    void* q = nullptr;
    cudaError_t e = cudaMalloc(&q, count * sizeof(T));
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        *p = nullptr;
        return map_cuda(e);
    }
    *p = static_cast<T*>(q);
    if (acc) *acc += count * sizeof(T);
    return FSP_OK;
}

// exp(-2 pi i m / L) evaluated in long double with exact octant symmetry
double2 unit_root(long m, long L) {
    const long double PI2 = 6.283185307179586476925286766559005768L;
    m %= L;
    // reduce to the first octant so that e.g. m = L/8 gives equal re/im and m = L/4 gives exactly -i
    long double c, s, a;
    const int q = (int)((8LL * m) / L);  // octant 0..7
    switch (q) {
        case 0: a = PI2 * m / L; c = cosl(a); s = sinl(a); break;
        case 1: a = PI2 * (L / 4.0L - m) / L; c = sinl(a); s = cosl(a); break;
        case 2: a = PI2 * (m - L / 4.0L) / L; c = -sinl(a); s = cosl(a); break;
        case 3: a = PI2 * (L / 2.0L - m) / L; c = -cosl(a); s = sinl(a); break;
        case 4: a = PI2 * (m - L / 2.0L) / L; c = -cosl(a); s = -sinl(a); break;
        case 5: a = PI2 * (3.0L * L / 4.0L - m) / L; c = -sinl(a); s = -cosl(a); break;
        case 6: a = PI2 * (m - 3.0L * L / 4.0L) / L; c = sinl(a); s = -cosl(a); break;
        default: a = PI2 * (L - m) / (long double)L; c = cosl(a); s = -sinl(a); break;
    }
    return make_double2((double)c, (double)(-s));
}

int upload_table(double2** dst, const std::vector<double2>& hst, size_t* acc) {
    int rc = dev_alloc(dst, hst.size(), acc);
    if (rc != FSP_OK) return rc;
    CU(cudaMemcpy(*dst, hst.data(), sizeof(double2) * hst.size(), cudaMemcpyHostToDevice));
    return FSP_OK;
}

// exp(-2 pi i n / L), n < L
int make_table(double2** dst, int L, size_t* acc) {
    std::vector<double2> hst((size_t)L);
    for (int n = 0; n < L; ++n) hst[n] = unit_root(n, L);
    return upload_table(dst, hst, acc);
}

// (cos, tan) of exp(-2 pi i m / L) in long double; an exactly vanishing cosine is replaced by 2^-200 so
// that c * (x + y * (s/c)) still evaluates to s * y (fft_warp.cuh dft_lane, "tan form")
void cos_tan(long m, long L, double* c_out, double* t_out) {
    const long double PI2 = 6.283185307179586476925286766559005768L;
    m %= L;
    long double c, s;
    if (4 * m == L) { c = 0.0L; s = 1.0L; }
    else if (2 * m == L) { c = -1.0L; s = 0.0L; }
    else if (4 * m == 3 * L) { c = 0.0L; s = -1.0L; }
    else if (m == 0) { c = 1.0L; s = 0.0L; }
    else { const long double a = PI2 * (long double)m / (long double)L; c = cosl(a); s = sinl(a); }
    if (c == 0.0L) c = ldexpl(1.0L, -200);
    *c_out = (double)c;
    *t_out = (double)(s / c);
}

// lane-constant stage-2 twiddles of fft_warp.cuh: for butterfly j < R1, level r = 2,4,..,R2, k < max(1,r/4):
//   b_r w_r^k = exp(-2 pi i (j R2 + k M) / (r M)),  stored as [j][cos(NC) | tan(NC)], index r/4 + k (level 2: 0)
int make_lane_table(double** dst, int M, int R1, size_t* acc) {
    const int R2 = M / R1, NC = R2 >= 4 ? R2 / 2 : 1;
    std::vector<double> hst((size_t)R1 * 2 * NC, 0.0);
    for (int j = 0; j < R1; ++j)
        for (int r = 2; r <= R2; r *= 2) {
            const int ofs = r >= 4 ? r / 4 : 0, q = r >= 4 ? r / 4 : 1;
            for (int k = 0; k < q; ++k)
                cos_tan((long)j * R2 + (long)k * M, (long)r * M, &hst[(size_t)j * 2 * NC + ofs + k],
                        &hst[(size_t)j * 2 * NC + NC + ofs + k]);
        }
    int rc = dev_alloc(dst, hst.size(), acc);
    if (rc != FSP_OK) return rc;
    CU(cudaMemcpy(*dst, hst.data(), sizeof(double) * hst.size(), cudaMemcpyHostToDevice));
    return FSP_OK;
}

template <int M>
int lane_table_for(double** dst, size_t* acc) { return make_lane_table(dst, M, Fft2Cfg<M>::R1, acc); }

// constants of fft512s_forward (fft_warp.cuh): the stage-2 table of make_lane_table for 512 = 32 x 16, followed by
// (cos[8] | tan[8]) of w_32^(m + 8 h), m < 8, for h = 0 and h = 1 (the radix-2 level shared by lane pairs)
int make_lane_table_512s(double** dst, size_t* acc) {
    const int M = 512, R1 = 32, R2 = 16, NC = 8;
    std::vector<double> hst((size_t)R1 * 2 * NC + 32, 0.0);
    for (int j = 0; j < R1; ++j)
        for (int r = 2; r <= R2; r *= 2) {
            const int ofs = r >= 4 ? r / 4 : 0, q = r >= 4 ? r / 4 : 1;
            for (int k = 0; k < q; ++k)
                cos_tan((long)j * R2 + (long)k * M, (long)r * M, &hst[(size_t)j * 2 * NC + ofs + k],
                        &hst[(size_t)j * 2 * NC + NC + ofs + k]);
        }
    for (int h = 0; h < 2; ++h)
        for (int m = 0; m < 8; ++m)
            cos_tan(m + 8 * h, 32, &hst[(size_t)R1 * 2 * NC + h * 16 + m], &hst[(size_t)R1 * 2 * NC + h * 16 + 8 + m]);
    int rc = dev_alloc(dst, hst.size(), acc);
    if (rc != FSP_OK) return rc;
    CU(cudaMemcpy(*dst, hst.data(), sizeof(double) * hst.size(), cudaMemcpyHostToDevice));
    return FSP_OK;
}

// ---- TMA tensor maps ---------------------------------------------------------------------------------
// cuTensorMapEncodeTiled is fetched through the runtime so that libfsp.so does not link libcuda directly.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* q = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &q, cudaEnableDefault, &qr) != cudaSuccess ||
            qr != cudaDriverEntryPointSuccess) {
            (void)cudaGetLastError();
            return nullptr;
        }
        fn = reinterpret_cast<EncodeTiledFn>(q);
    }
    return fn;
}
// fp64 tensor of `rank` dimensions (dims[0] fastest, strides in bytes for dims 1..rank-1), no swizzle
int make_tensor_map(CUtensorMap* tm, void* base, int rank, const cuuint64_t* dims, const cuuint64_t* strides,
                    const cuuint32_t* box) {
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return FSP_ERR_CUDA;
    cuuint32_t es[5] = {1, 1, 1, 1, 1};
    CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, (cuuint32_t)rank, base, dims, strides, box, es,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? FSP_OK : FSP_ERR_CUDA;
}

// ---- per-device caches -------------------------------------------------------------------------------
// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) and the occupancy of a kernel belong to a DEVICE, not to the
// process: every launch helper keeps one slot per device (zero = not yet queried; the query is idempotent, so two
// host threads racing on a slot do no harm).
constexpr int kMaxDevices = 64;
struct OccCache { std::atomic<int> v[kMaxDevices]; };
template <class Kern>
int cached_occupancy(OccCache& c, int dev, Kern kern, int threads, size_t smem, int* occ_out) {
    int o = c.v[dev].load(std::memory_order_acquire);
    if (o == 0) {
        CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, kern, threads, smem));
        if (o < 1) return FSP_ERR_CUDA;
        c.v[dev].store(o, std::memory_order_release);
    }
    *occ_out = o;
    return FSP_OK;
}
// shared-memory opt-in of a precompute kernel whose request varies with the transform length: raised only when a launch
// needs more than any earlier one on this device (setting the attribute before every launch costs milliseconds)
template <class Kern>
int cached_smem_optin(OccCache& c, int dev, Kern kern, size_t smem) {
    if (c.v[dev].load(std::memory_order_acquire) < (int)smem) {
        CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        c.v[dev].store((int)smem, std::memory_order_release);
    }
    return FSP_OK;
}

// Every entry point runs on the plan's device and restores the caller's current device on return.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
};

// ---- kernel launch helpers (one template instantiation per FFT length) ---------------------------
template <int M>
int launch_fwd_y_t(fsp_plan* p, int kx0, double2* B2, int nplanes) {
    using Y = TileY<M>;
    const long ntiles = (long)nplanes * (p->Nz / Y::KW);
    const size_t smem = Y::smem_bytes();
    static OccCache cache;   // per device: function attributes and occupancy belong to the device
    int occ = 0;
    { const int rc_ = cached_occupancy(cache, p->device, k_fwd_y_t<M>, Y::THREADS, smem, &occ); if (rc_ != FSP_OK) return rc_; }
    long grid = (long)p->sm_count * occ;
    if (grid > ntiles) grid = ntiles;
    k_fwd_y_t<M><<<(unsigned)grid, Y::THREADS, smem, p->stream>>>(p->tmB1y, B2, p->LTy, p->Wy, p->Nz, kx0, ntiles);
    return FSP_OK;
}
template <int M2>
int launch_fwd_y_f(fsp_plan* p, int kx0, double2* B2, int nplanes) {
    using Y = TileYF<M2>;
    const long ntiles = (long)nplanes * (p->Nz / Y::KW);
    const size_t smem = Y::smem_bytes();
    static OccCache cache;
    int occ = 0;
    { const int rc_ = cached_occupancy(cache, p->device, k_fwd_y_f<M2>, Y::THREADS, smem, &occ); if (rc_ != FSP_OK) return rc_; }
    long grid = (long)p->sm_count * occ;
    if (grid > ntiles) grid = ntiles;
    k_fwd_y_f<M2><<<(unsigned)grid, Y::THREADS, smem, p->stream>>>(p->tmB1y, B2, p->LTyf, p->Nz, kx0, ntiles);
    return FSP_OK;
}
template <int M>
int launch_fwd_y(fsp_plan* p, const double2* B1, double2* B2, int nplanes) {
    using Cfg = FftCfg<M>;
    constexpr int G = TileGroups<Cfg>::G;
    const long ntiles = (long)nplanes * (p->Nz / kW);
    const size_t smem = sizeof(double2) * (size_t)(2 * M + G * M * kW);
    static OccCache cache;   // per device: function attributes and occupancy belong to the device
    int occ = 0;
    { const int rc_ = cached_occupancy(cache, p->device, k_fwd_y<M>, G * kW * Cfg::T, smem, &occ); if (rc_ != FSP_OK) return rc_; }
    long grid = (ntiles + G - 1) / G;
    if (grid > (long)p->sm_count * occ) grid = (long)p->sm_count * occ;
    k_fwd_y<M><<<(unsigned)grid, G * kW * Cfg::T, smem, p->stream>>>(B1, B2, p->Wy, p->Nz, ntiles);
    return FSP_OK;
}
template <int M, bool DER>
int launch_inv_y_impl(fsp_plan* p, const double2* B2, double2* B1, int nplanes, double kder) {
    using Cfg = FftCfg<M>;
    constexpr int G = TileGroups<Cfg>::G;
    const long ntiles = (long)nplanes * (p->Nz / kW);
    const size_t smem = sizeof(double2) * (size_t)(2 * M + G * M * kW);
    static OccCache cache;   // per device: function attributes and occupancy belong to the device
    int occ = 0;
    { const int rc_ = cached_occupancy(cache, p->device, k_inv_y<M, DER>, G * kW * Cfg::T, smem, &occ); if (rc_ != FSP_OK) return rc_; }
    long grid = (ntiles + G - 1) / G;
    if (grid > (long)p->sm_count * occ) grid = (long)p->sm_count * occ;
    k_inv_y<M, DER><<<(unsigned)grid, G * kW * Cfg::T, smem, p->stream>>>(B2, B1, p->Wy, p->Nz, ntiles, kder);
    return FSP_OK;
}
// kder != 0: the E_y variant (input rows times -i kder m'(ky))
template <int M>
int launch_inv_y(fsp_plan* p, const double2* B2, double2* B1, int nplanes, double kder) {
    return kder != 0.0 ? launch_inv_y_impl<M, true>(p, B2, B1, nplanes, kder) : launch_inv_y_impl<M, false>(p, B2, B1, nplanes, 0.0);
}
// DER = false: in place on B2.  DER = true: B2 -> out with the factor -i k_d of `kap` (field output).
template <int M, bool DER>
int launch_conv_z_p_impl(fsp_plan* p, double2* B2, const double* G, int nplanes, double2* out, const DerK kap) {
    using Z = ConvZP<M>;
    const long nsteps = (long)nplanes * (2 * p->Ny) / Z::G;   // pair steps: G pencils each
    const size_t smem = Z::smem_bytes();
    static OccCache cache;   // per device: function attributes and occupancy belong to the device
    int occ = 0;
    { const int rc_ = cached_occupancy(cache, p->device, k_conv_z_p<M, DER>, Z::WARPS * 32, smem, &occ); if (rc_ != FSP_OK) return rc_; }
    long grid = (long)p->sm_count * occ;
    const long need = (nsteps + Z::PAIRS - 1) / Z::PAIRS;
    if (grid > need) grid = need;
    k_conv_z_p<M, DER><<<(unsigned)grid, Z::WARPS * 32, smem, p->stream>>>(B2, G, p->LTz, p->Wz, p->Ny, nsteps, out, kap);
    return FSP_OK;
}
template <bool DER>
int launch_conv_z_s_impl(fsp_plan* p, double2* B2, const double* G, int nplanes, double2* out, const DerK kap) {
    using Z = ConvZS;
    const long nsteps = (long)nplanes * (2 * p->Ny);   // pair steps: one pencil each
    const size_t smem = Z::smem_bytes();
    static OccCache cache;   // per device: function attributes and occupancy belong to the device
    int occ = 0;
    { const int rc_ = cached_occupancy(cache, p->device, k_conv_z_s<DER>, Z::WARPS * 32, smem, &occ); if (rc_ != FSP_OK) return rc_; }
    long grid = (long)p->sm_count * occ;
    const long need = (nsteps + Z::PAIRS - 1) / Z::PAIRS;
    if (grid > need) grid = need;
    k_conv_z_s<DER><<<(unsigned)grid, Z::WARPS * 32, smem, p->stream>>>(B2, G, p->LTzs, p->Wz, p->Ny, nsteps, out, kap);
    return FSP_OK;
}
template <int M2, bool DER>
int launch_conv_z_f_impl(fsp_plan* p, double2* B2, const double* G, int nplanes, double2* out, const DerK kap) {
    using Z = ConvZF<M2>;
    const long ngroups = (long)nplanes * (2 * p->Ny) / Z::G;
    const size_t smem = Z::smem_bytes();
    static OccCache cache;   // per device: function attributes and occupancy belong to the device
    int occ = 0;
    { const int rc_ = cached_occupancy(cache, p->device, k_conv_z_f<M2, DER>, Z::WARPS * 32, smem, &occ); if (rc_ != FSP_OK) return rc_; }
    long grid = (long)p->sm_count * occ;
    const long need = (ngroups + Z::WARPS - 1) / Z::WARPS;
    if (grid > need) grid = need;
    k_conv_z_f<M2, DER><<<(unsigned)grid, Z::WARPS * 32, smem, p->stream>>>(B2, G, p->LTzf, p->Ny, ngroups, out, kap);
    return FSP_OK;
}
template <int M, bool DER>
int launch_conv_z_w_impl(fsp_plan* p, double2* B2, const double* G, int nplanes, double2* out, const DerK kap) {
    // Nz = 256, 512: the whole padded pencil in one lane group (k_conv_z_f); FSP_PARAM_K3_VARIANT = 1 and Nz = 1024:
    // warp pairs (k_conv_z_p); variant 2 at Nz = 512: warp pairs with 32 lanes per branch (k_conv_z_s);
    // below 256: both branches in one warp (k_conv_z_w)
    if constexpr (M == 512 || M == 256) { if (p->gk_natural) return launch_conv_z_f_impl<2 * M, DER>(p, B2, G, nplanes, out, kap); }
    if constexpr (M == 512) { if (p->k3_variant == 2) return launch_conv_z_s_impl<DER>(p, B2, G, nplanes, out, kap); }
    if constexpr (M >= 256) return launch_conv_z_p_impl<M, DER>(p, B2, G, nplanes, out, kap);
    else {
    using Z = ConvZ<M>;
    const long ngroups = (long)nplanes * (2 * p->Ny) / Z::G;
    const size_t smem = Z::smem_bytes();
    static OccCache cache;   // per device: function attributes and occupancy belong to the device
    int occ = 0;
    { const int rc_ = cached_occupancy(cache, p->device, k_conv_z_w<M, DER>, Z::WARPS * 32, smem, &occ); if (rc_ != FSP_OK) return rc_; }
    long grid = (long)p->sm_count * occ;
    const long need = (ngroups + Z::WARPS - 1) / Z::WARPS;
    if (grid > need) grid = need;
    k_conv_z_w<M, DER><<<(unsigned)grid, Z::WARPS * 32, smem, p->stream>>>(B2, G, p->LTz, p->Wz, p->Ny, ngroups, out, kap);
    return FSP_OK;
    }
}
template <int M>
int launch_conv_z_w(fsp_plan* p, double2* B2, const double* G, int nplanes, double2* out, const DerK* kap) {
    if (kap) return launch_conv_z_w_impl<M, true>(p, B2, G, nplanes, out, *kap);
    return launch_conv_z_w_impl<M, false>(p, B2, G, nplanes, nullptr, DerK{0.0, 0.0, 0.0, 0});
}
template <int M>
int launch_fwd_x(fsp_plan* p, const double* rho) {
    using Cfg = FftCfg<M>;
    constexpr int G = TileGroups<Cfg>::G;
    const long ntiles = (long)p->Ny * (p->Nz / kW);
    const size_t smem = sizeof(double2) * (size_t)(4 * M + G * M * kW + G * 2 * M * kW);
    static OccCache cache;
    int occ = 0;
    { const int rc_ = cached_occupancy(cache, p->device, k_fwd_x_r2c<M>, G * kW * Cfg::T, smem, &occ); if (rc_ != FSP_OK) return rc_; }
    k_fwd_x_r2c<M><<<(unsigned)((ntiles + G - 1) / G), G * kW * Cfg::T, smem, p->stream>>>(rho, p->B1, p->Wx, p->Ny, p->Nz, ntiles);
    return FSP_OK;
}
template <int M, bool DER>
int launch_inv_x_impl(fsp_plan* p, double* phi, double kder) {
    using Cfg = FftCfg<M>;
    constexpr int G = TileGroups<Cfg>::G;
    const long ntiles = (long)p->Ny * (p->Nz / kW);
    const size_t smem = sizeof(double2) * (size_t)(4 * M + G * M * kW);
    static OccCache cache;
    int occ = 0;
    { const int rc_ = cached_occupancy(cache, p->device, k_inv_x_c2r<M, DER>, G * kW * Cfg::T, smem, &occ); if (rc_ != FSP_OK) return rc_; }
    k_inv_x_c2r<M, DER><<<(unsigned)((ntiles + G - 1) / G), G * kW * Cfg::T, smem, p->stream>>>(p->B1, phi, p->Wx, p->Ny, p->Nz, ntiles, kder);
    return FSP_OK;
}
// kder != 0: the E_x variant (X[k] times -i kder k)
template <int M>
int launch_inv_x(fsp_plan* p, double* phi, double kder) {
    return kder != 0.0 ? launch_inv_x_impl<M, true>(p, phi, kder) : launch_inv_x_impl<M, false>(p, phi, 0.0);
}

#define DISPATCH_YZ(fn, M, ...)                          \
    switch (M) {                                         \
        case 12: return fn<12>(__VA_ARGS__);             \
        case 24: return fn<24>(__VA_ARGS__);             \
        case 48: return fn<48>(__VA_ARGS__);             \
        case 96: return fn<96>(__VA_ARGS__);             \
        case 192: return fn<192>(__VA_ARGS__);           \
        case 384: return fn<384>(__VA_ARGS__);           \
        case 768: return fn<768>(__VA_ARGS__);           \
        case 20: return fn<20>(__VA_ARGS__);             \
        case 40: return fn<40>(__VA_ARGS__);             \
        case 80: return fn<80>(__VA_ARGS__);             \
        case 160: return fn<160>(__VA_ARGS__);           \
        case 320: return fn<320>(__VA_ARGS__);           \
        case 8: return fn<8>(__VA_ARGS__);               \
        case 16: return fn<16>(__VA_ARGS__);             \
        case 32: return fn<32>(__VA_ARGS__);             \
        case 64: return fn<64>(__VA_ARGS__);             \
        case 128: return fn<128>(__VA_ARGS__);           \
        case 256: return fn<256>(__VA_ARGS__);           \
        case 512: return fn<512>(__VA_ARGS__);           \
        case 1024: return fn<1024>(__VA_ARGS__);         \
        default: return FSP_ERR_INVALID_ARG;             \
    }
#define DISPATCH_X(fn, M, ...)                           \
    switch (M) {                                         \
        case 6: return fn<6>(__VA_ARGS__);               \
        case 12: return fn<12>(__VA_ARGS__);             \
        case 24: return fn<24>(__VA_ARGS__);             \
        case 48: return fn<48>(__VA_ARGS__);             \
        case 96: return fn<96>(__VA_ARGS__);             \
        case 192: return fn<192>(__VA_ARGS__);           \
        case 384: return fn<384>(__VA_ARGS__);           \
        case 10: return fn<10>(__VA_ARGS__);             \
        case 20: return fn<20>(__VA_ARGS__);             \
        case 40: return fn<40>(__VA_ARGS__);             \
        case 80: return fn<80>(__VA_ARGS__);             \
        case 160: return fn<160>(__VA_ARGS__);           \
        case 4: return fn<4>(__VA_ARGS__);               \
        case 8: return fn<8>(__VA_ARGS__);               \
        case 16: return fn<16>(__VA_ARGS__);             \
        case 32: return fn<32>(__VA_ARGS__);             \
        case 64: return fn<64>(__VA_ARGS__);             \
        case 128: return fn<128>(__VA_ARGS__);           \
        case 256: return fn<256>(__VA_ARGS__);           \
        case 512: return fn<512>(__VA_ARGS__);           \
        default: return FSP_ERR_INVALID_ARG;             \
    }

template <int M>
int launch_fwd_x_t(fsp_plan* p) {
    using X_ = TileX<M>;
    const long plane = (long)p->Ny * p->Nz, ntiles = plane / X_::KC;
    const size_t smem = X_::smem_bytes();
    static OccCache cache;   // per device: function attributes and occupancy belong to the device
    int occ = 0;
    { const int rc_ = cached_occupancy(cache, p->device, k_fwd_x_t<M>, X_::THREADS, smem, &occ); if (rc_ != FSP_OK) return rc_; }
    long grid = (long)p->sm_count * occ;
    if (grid > ntiles) grid = ntiles;
    k_fwd_x_t<M><<<(unsigned)grid, X_::THREADS, smem, p->stream>>>(p->tmRho, p->B1, p->LTx, p->Wx, plane, ntiles);
    return FSP_OK;
}
int do_fwd_x(fsp_plan* p, const double* rho) {
    if (p->tile_x && (reinterpret_cast<uintptr_t>(rho) & 15) == 0) {
        if (rho != p->tmRho_ptr) {   // the caller owns rho: encode the map for this address (host only, ~1 us)
            const cuuint64_t dims[2] = {(cuuint64_t)p->Ny * p->Nz, (cuuint64_t)p->Nx};
            const cuuint64_t strides[1] = {(cuuint64_t)p->Ny * p->Nz * 8};
            const cuuint32_t box[2] = {(cuuint32_t)(p->Nx == 1024 ? 8 : kC), (cuuint32_t)(p->Nx < 256 ? p->Nx : 256)};   // TileX<M>::KC columns
            int rc = make_tensor_map(&p->tmRho, const_cast<double*>(rho), 2, dims, strides, box);
            if (rc != FSP_OK) return rc;
            p->tmRho_ptr = rho;
        }
        if (p->Nx == 1024) return launch_fwd_x_t<512>(p);
        if (p->Nx == 512) return launch_fwd_x_t<256>(p);
        if (p->Nx == 256) return launch_fwd_x_t<128>(p);
        return launch_fwd_x_t<64>(p);
    }
    DISPATCH_X(launch_fwd_x, p->Nx / 2, p, rho)
}
int do_fwd_y(fsp_plan* p, int kx0, double2* B2, int np) {
    if (p->tile_y) {
        if (p->Ny == 1024) return launch_fwd_y_t<1024>(p, kx0, B2, np);
        if (p->Ny == 512 && p->k2_variant == 0) return launch_fwd_y_f<1024>(p, kx0, B2, np);
        if (p->Ny == 512) return launch_fwd_y_t<512>(p, kx0, B2, np);
        if (p->Ny == 256) return launch_fwd_y_t<256>(p, kx0, B2, np);
        return launch_fwd_y_t<128>(p, kx0, B2, np);
    }
    const double2* B1 = p->B1 + (size_t)kx0 * p->Ny * p->Nz;
    DISPATCH_YZ(launch_fwd_y, p->Ny, p, B1, B2, np)
}
#define DISPATCH_W(fn, M, ...)                           \
    switch (M) {                                         \
        case 8: return fn<8>(__VA_ARGS__);               \
        case 16: return fn<16>(__VA_ARGS__);             \
        case 32: return fn<32>(__VA_ARGS__);             \
        case 64: return fn<64>(__VA_ARGS__);             \
        case 128: return fn<128>(__VA_ARGS__);           \
        case 256: return fn<256>(__VA_ARGS__);           \
        case 512: return fn<512>(__VA_ARGS__);           \
        case 1024: return fn<1024>(__VA_ARGS__);         \
        default: return FSP_ERR_INVALID_ARG;             \
    }
template <int M, bool DER>
int launch_conv_z_g_impl(fsp_plan* p, double2* B2, const double* G, int nplanes, double2* out, const DerK kap) {
    using Cfg = FftCfg<M>;
    constexpr int GT = TileGroups<Cfg>::G;
    const long npencils = (long)nplanes * (2 * p->Ny);
    const size_t smem = sizeof(double2) * (size_t)(2 * M + GT * M * kW);
    static OccCache cache;
    int occ = 0;
    { const int rc_ = cached_occupancy(cache, p->device, k_conv_z_g<M, DER>, GT * kW * Cfg::T, smem, &occ); if (rc_ != FSP_OK) return rc_; }
    long grid = (npencils + (long)GT * kW - 1) / ((long)GT * kW);
    if (grid > (long)p->sm_count * occ) grid = (long)p->sm_count * occ;
    k_conv_z_g<M, DER><<<(unsigned)grid, GT * kW * Cfg::T, smem, p->stream>>>(B2, G, p->Wz, p->Ny, npencils, out, kap);
    return FSP_OK;
}
template <int M>
int launch_conv_z_g(fsp_plan* p, double2* B2, const double* G, int np, double2* out, const DerK* kap) {
    if (kap) return launch_conv_z_g_impl<M, true>(p, B2, G, np, out, *kap);
    return launch_conv_z_g_impl<M, false>(p, B2, G, np, nullptr, DerK{0.0, 0.0, 0.0, 0});
}
template <int M2, bool DER>
int launch_conv_z_g2_impl(fsp_plan* p, double2* B2, const double* G, int nplanes, double2* out, const DerK kap) {
    using Cfg = FftCfg<M2>;
    constexpr int GT = TileGroups<Cfg>::G;
    const long npencils = (long)nplanes * (2 * p->Ny);
    const size_t smem = sizeof(double2) * (size_t)(M2 + GT * M2 * kW);
    static OccCache cache;
    int occ = 0;
    { const int rc_ = cached_occupancy(cache, p->device, k_conv_z_g2<M2, DER>, GT * kW * Cfg::T, smem, &occ); if (rc_ != FSP_OK) return rc_; }
    long grid = (npencils + (long)GT * kW - 1) / ((long)GT * kW);
    if (grid > (long)p->sm_count * occ) grid = (long)p->sm_count * occ;
    k_conv_z_g2<M2, DER><<<(unsigned)grid, GT * kW * Cfg::T, smem, p->stream>>>(B2, G, p->Wz, p->Ny, npencils, out, kap);
    return FSP_OK;
}
template <int M2>
int launch_conv_z_g2(fsp_plan* p, double2* B2, const double* G, int np, double2* out, const DerK* kap) {
    if (kap) return launch_conv_z_g2_impl<M2, true>(p, B2, G, np, out, *kap);
    return launch_conv_z_g2_impl<M2, false>(p, B2, G, np, nullptr, DerK{0.0, 0.0, 0.0, 0});
}
template <int B, int P, bool DER>
int launch_conv_z_pf_impl(fsp_plan* p, double2* B2, const double* G, int nplanes, double2* out, const DerK kap) {
    using Z = ConvZPF<B, P>;
    const long ngroups = (long)nplanes * (2 * p->Ny) / Z::G;
    const size_t smem = Z::smem_bytes();
    static OccCache cache;
    int occ = 0;
    { const int rc_ = cached_occupancy(cache, p->device, k_conv_z_pf<B, P, DER>, Z::WARPS * 32, smem, &occ); if (rc_ != FSP_OK) return rc_; }
    long grid = (long)p->sm_count * occ;
    const long need = (ngroups + Z::WARPS - 1) / Z::WARPS;
    if (grid > need) grid = need;
    k_conv_z_pf<B, P, DER><<<(unsigned)grid, Z::WARPS * 32, smem, p->stream>>>(B2, G, p->LTzf, p->Ny, ngroups, out, kap);
    return FSP_OK;
}
template <int B, int P>
int launch_conv_z_pf(fsp_plan* p, double2* B2, const double* G, int np, double2* out, const DerK* kap) {
    if (kap) return launch_conv_z_pf_impl<B, P, true>(p, B2, G, np, out, *kap);
    return launch_conv_z_pf_impl<B, P, false>(p, B2, G, np, nullptr, DerK{0.0, 0.0, 0.0, 0});
}
bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }
// Nz = 3 * 2^k, 5 * 2^k with a warp-level prime-factor kernel (2 Nz = B P, B = 3: P = 16 .. 256, B = 5: P = 16 .. 64)
// (Nz = 320 would need 5 x 16 complex registers per lane and 233 KB of shared memory, Nz = 768 3 x 32: CTA-level kernel)
bool z_uses_pf(int Nz) { return Nz == 24 || Nz == 48 || Nz == 96 || Nz == 192 || Nz == 384 || Nz == 40 || Nz == 80 || Nz == 160; }
int pf_radix(int Nz) { return Nz % 3 == 0 ? 3 : 5; }
// doubles per spectrum row as ALLOCATED: Nz + 2 (octant rows, natural or [E | O]); 2 Nz where the prime-factor kernel may run
size_t gk_row(int Nz) { return z_uses_pf(Nz) ? (size_t)2 * Nz : (size_t)Nz + 2; }
// Nz = 3 * 2^k, 5 * 2^k whose doubled length has an engine configuration: k_conv_z_g2 (natural-order spectrum rows)
bool z_uses_g2(int Nz) { return Nz == 24 || Nz == 48 || Nz == 96 || Nz == 192 || Nz == 384 || Nz == 40 || Nz == 80 || Nz == 160; }
int do_conv_z_w(fsp_plan* p, double2* B2, const double* G, int np, double2* out, const DerK* kap) {
    if (!is_pow2(p->Nz)) {   // 3 * 2^k, 5 * 2^k: the prime-factor warp kernel, else the CTA-level kernels on the mixed-radix engine
        if (p->gk_pfa) {
            switch (p->Nz) {
                case 384: return launch_conv_z_pf<3, 256>(p, B2, G, np, out, kap);
                case 192: return launch_conv_z_pf<3, 128>(p, B2, G, np, out, kap);
                case 96: return launch_conv_z_pf<3, 64>(p, B2, G, np, out, kap);
                case 48: return launch_conv_z_pf<3, 32>(p, B2, G, np, out, kap);
                case 24: return launch_conv_z_pf<3, 16>(p, B2, G, np, out, kap);
                case 160: return launch_conv_z_pf<5, 64>(p, B2, G, np, out, kap);
                case 80: return launch_conv_z_pf<5, 32>(p, B2, G, np, out, kap);
                case 40: return launch_conv_z_pf<5, 16>(p, B2, G, np, out, kap);
                default: return FSP_ERR_INVALID_ARG;
            }
        }
        if (p->gk_natural) {
            switch (p->Nz) {
                case 24: return launch_conv_z_g2<48>(p, B2, G, np, out, kap);
                case 48: return launch_conv_z_g2<96>(p, B2, G, np, out, kap);
                case 96: return launch_conv_z_g2<192>(p, B2, G, np, out, kap);
                case 192: return launch_conv_z_g2<384>(p, B2, G, np, out, kap);
                case 384: return launch_conv_z_g2<768>(p, B2, G, np, out, kap);
                case 40: return launch_conv_z_g2<80>(p, B2, G, np, out, kap);
                case 80: return launch_conv_z_g2<160>(p, B2, G, np, out, kap);
                case 160: return launch_conv_z_g2<320>(p, B2, G, np, out, kap);
                default: return FSP_ERR_INVALID_ARG;
            }
        }
        switch (p->Nz) {
            case 12: return launch_conv_z_g<12>(p, B2, G, np, out, kap);
            case 24: return launch_conv_z_g<24>(p, B2, G, np, out, kap);
            case 48: return launch_conv_z_g<48>(p, B2, G, np, out, kap);
            case 96: return launch_conv_z_g<96>(p, B2, G, np, out, kap);
            case 192: return launch_conv_z_g<192>(p, B2, G, np, out, kap);
            case 384: return launch_conv_z_g<384>(p, B2, G, np, out, kap);
            case 768: return launch_conv_z_g<768>(p, B2, G, np, out, kap);
            case 20: return launch_conv_z_g<20>(p, B2, G, np, out, kap);
            case 40: return launch_conv_z_g<40>(p, B2, G, np, out, kap);
            case 80: return launch_conv_z_g<80>(p, B2, G, np, out, kap);
            case 160: return launch_conv_z_g<160>(p, B2, G, np, out, kap);
            case 320: return launch_conv_z_g<320>(p, B2, G, np, out, kap);
            default: return FSP_ERR_INVALID_ARG;
        }
    }
    DISPATCH_W(launch_conv_z_w, p->Nz, p, B2, G, np, out, kap)
}
// planes [kx0, kx0 + np) of the spectrum go with the np planes stored at B2.
// kap == nullptr: in place (phi); otherwise B2 -> out with the derivative factor (whole volume only, kx0 = 0).
// periodic z (FSP_PARAM_PERIODIC bit 4) on power-of-two Nz: Nz-point transforms instead of the padded 2 Nz (k_conv_z_periodic)
template <int M, bool NATURAL>
int launch_conv_z_periodic_impl(fsp_plan* p, double2* B2, const double* G, int nplanes) {
    using Z = ConvZPer<M>;
    const long npencils = (long)nplanes * (2 * p->Ny), ngroups = (npencils + Z::G - 1) / Z::G;
    const size_t smem = Z::smem_bytes();
    static OccCache cache;
    int occ = 0;
    { const int rc_ = cached_occupancy(cache, p->device, k_conv_z_periodic<M, NATURAL>, Z::WARPS * 32, smem, &occ); if (rc_ != FSP_OK) return rc_; }
    long grid = (long)p->sm_count * occ;
    const long need = (ngroups + Z::WARPS - 1) / Z::WARPS;
    if (grid > need) grid = need;
    k_conv_z_periodic<M, NATURAL><<<(unsigned)grid, Z::WARPS * 32, smem, p->stream>>>(B2, G, p->LTz, p->Ny, ngroups, npencils);
    CU(cudaGetLastError());
    return FSP_OK;
}
template <int M>
int launch_conv_z_periodic(fsp_plan* p, double2* B2, const double* G, int nplanes) {
    // natural-order rows exist where k_conv_z_f runs (Nz = 256, 512), [E | O] rows elsewhere
    if constexpr (M == 256 || M == 512) {
        if (p->gk_natural) return launch_conv_z_periodic_impl<M, true>(p, B2, G, nplanes);
    }
    if (p->gk_natural) return FSP_ERR_INVALID_ARG;
    return launch_conv_z_periodic_impl<M, false>(p, B2, G, nplanes);
}
int do_conv_z(fsp_plan* p, double2* B2, int kx0, int np, double2* out = nullptr, const DerK* kap = nullptr) {
    if ((p->periodic & 4) && p->periodic_fast_z && !out && !kap && !p->gk_pfa && is_pow2(p->Nz) && p->LTz) {
        const double* G = p->Gk + (size_t)kx0 * (p->Ny + 1) * ((size_t)p->Nz + 2);
        switch (p->Nz) {
            case 8: return launch_conv_z_periodic<8>(p, B2, G, np);
            case 16: return launch_conv_z_periodic<16>(p, B2, G, np);
            case 32: return launch_conv_z_periodic<32>(p, B2, G, np);
            case 64: return launch_conv_z_periodic<64>(p, B2, G, np);
            case 128: return launch_conv_z_periodic<128>(p, B2, G, np);
            case 256: return launch_conv_z_periodic<256>(p, B2, G, np);
            case 512: return launch_conv_z_periodic<512>(p, B2, G, np);
            case 1024: return launch_conv_z_periodic<1024>(p, B2, G, np);
            default: break;
        }
    }
    return do_conv_z_w(p, B2, p->Gk + (size_t)kx0 * (p->Ny + 1) * (p->gk_pfa ? (size_t)2 * p->Nz : (size_t)p->Nz + 2), np, out, kap);
}
int make_z_lane_table(fsp_plan* p) {
    if (!is_pow2(p->Nz)) return FSP_OK;   // k_conv_z_g reads the root table only
    DISPATCH_W(lane_table_for, p->Nz, &p->LTz, &p->bytes)
}
int make_x_lane_table(fsp_plan* p) { DISPATCH_W(lane_table_for, p->Nx / 2, &p->LTx, &p->bytes) }
int make_y_lane_table(fsp_plan* p) { DISPATCH_W(lane_table_for, p->Ny, &p->LTy, &p->bytes) }
template <int M, bool DER>
int launch_inv_y_t_impl(fsp_plan* p, const CUtensorMap& tm, double2* B1, int nplanes, double kder) {
    using Y = TileYI<M>;
    const long ntiles = (long)nplanes * (p->Nz / Y::KW);
    const size_t smem = Y::smem_bytes();
    static OccCache cache;   // per device: function attributes and occupancy belong to the device
    int occ = 0;
    { const int rc_ = cached_occupancy(cache, p->device, k_inv_y_t<M, DER>, Y::THREADS, smem, &occ); if (rc_ != FSP_OK) return rc_; }
    long grid = (long)p->sm_count * occ;
    if (grid > ntiles) grid = ntiles;
    k_inv_y_t<M, DER><<<(unsigned)grid, Y::THREADS, smem, p->stream>>>(tm, B1, p->LTy, p->Wy, p->Nz, ntiles, kder);
    return FSP_OK;
}
template <int M>
int launch_inv_y_t(fsp_plan* p, const CUtensorMap& tm, double2* B1, int nplanes, double kder) {
    return kder != 0.0 ? launch_inv_y_t_impl<M, true>(p, tm, B1, nplanes, kder) : launch_inv_y_t_impl<M, false>(p, tm, B1, nplanes, 0.0);
}
// B2 must be the plan's own B2 (the tile kernel reads it through the plan's tensor map)
int do_inv_y(fsp_plan* p, const double2* B2, double2* B1, int np, double kder = 0.0) {
    if (p->tile_y && (B2 == p->B2 || (p->B3 && B2 == p->B3))) {
        const CUtensorMap& tm = B2 == p->B2 ? p->tmB2y : p->tmB3y;
        if (p->Ny == 1024) return launch_inv_y_t<1024>(p, tm, B1, np, kder);
        if (p->Ny == 512) return launch_inv_y_t<512>(p, tm, B1, np, kder);
        if (p->Ny == 256) return launch_inv_y_t<256>(p, tm, B1, np, kder);
        return launch_inv_y_t<128>(p, tm, B1, np, kder);
    }
    DISPATCH_YZ(launch_inv_y, p->Ny, p, B2, B1, np, kder)
}
template <int M, bool DER>
int launch_inv_x_t_impl(fsp_plan* p, double* phi, double kder) {
    using X_ = TileXI<M>;
    const long plane = (long)p->Ny * p->Nz, ntiles = plane / X_::KC;
    const size_t smem = X_::smem_bytes();
    static OccCache cache;   // per device: function attributes and occupancy belong to the device
    int occ = 0;
    { const int rc_ = cached_occupancy(cache, p->device, k_inv_x_t<M, DER>, X_::THREADS, smem, &occ); if (rc_ != FSP_OK) return rc_; }
    long grid = (long)p->sm_count * occ;
    if (grid > ntiles) grid = ntiles;
    k_inv_x_t<M, DER><<<(unsigned)grid, X_::THREADS, smem, p->stream>>>(p->tmB1x, p->B1, phi, p->LTx, p->Wx, plane, ntiles, kder);
    return FSP_OK;
}
template <int M>
int launch_inv_x_t(fsp_plan* p, double* phi, double kder) {
    return kder != 0.0 ? launch_inv_x_t_impl<M, true>(p, phi, kder) : launch_inv_x_t_impl<M, false>(p, phi, 0.0);
}
int do_inv_x(fsp_plan* p, double* phi, double kder = 0.0) {
    // Nx = 1024: 8-column tiles would write phi in half lines (measured 11.9 ms against 9.5 ms for the
    // first-generation kernel at 1024^3), so K5 stays on the first-generation kernel there (K1 does not: 7.9 vs 12.6)
    if (p->tile_x && p->Nx != 1024) {
        if (p->Nx == 512) return launch_inv_x_t<256>(p, phi, kder);
        if (p->Nx == 256) return launch_inv_x_t<128>(p, phi, kder);
        return launch_inv_x_t<64>(p, phi, kder);
    }
    DISPATCH_X(launch_inv_x, p->Nx / 2, p, phi, kder)
}

// embed (dir = 0: small -> big) or crop (dir = 1: big -> small) a Ux x Uy x Uz block at the origin of an
// Nx x Ny x Nz array (non-power-of-two meshes, R19); the rest of the big array stays zero
__global__ void k_embed_crop(double* __restrict__ big, double* __restrict__ small_, int Uy, int Uz, int Ny, int Nz,
                             long total, int dir) {
    for (long o = blockIdx.x * (long)blockDim.x + threadIdx.x; o < total; o += (long)gridDim.x * blockDim.x) {
        const int z = (int)(o % Uz), y = (int)((o / Uz) % Uy);
        const long x = o / ((long)Uz * Uy);
        const long q = (x * Ny + y) * Nz + z;
        if (dir == 0) big[q] = small_[o];
        else small_[o] = big[q];
    }
}

unsigned grid_for(long total, int block) {
    long g = (total + block - 1) / block;
    const long cap = 148L * 32;
    return (unsigned)(g < cap ? (g > 0 ? g : 1) : cap);
}

size_t user_volume(const fsp_plan* p) { return (size_t)p->Ux * p->Uy * p->Uz; }
int embed_rho(fsp_plan* p, const double* rho_user) {   // rho_pad <- rho (its zero part was set at plan creation)
    const long tot = (long)user_volume(p);
    k_embed_crop<<<grid_for(tot, 256), 256, 0, p->stream>>>(p->rho_pad, const_cast<double*>(rho_user), p->Uy, p->Uz, p->Ny, p->Nz, tot, 0);
    CU(cudaGetLastError());
    return FSP_OK;
}
int crop_out(fsp_plan* p, double* dst_user) {          // dst <- phi_pad restricted to the caller's mesh
    const long tot = (long)user_volume(p);
    k_embed_crop<<<grid_for(tot, 256), 256, 0, p->stream>>>(p->phi_pad, dst_user, p->Uy, p->Uz, p->Ny, p->Nz, tot, 1);
    CU(cudaGetLastError());
    return FSP_OK;
}
int next_pow2_min8(int n) { int q = 8; while (q < n) q *= 2; return q; }
// smallest transform length >= n that has kernels: 2^k, 3 * 2^k, 5 * 2^k between 8 and 1024.
// pow2_only: the plain Vico-Greengard precompute (its 4N-point FFTs are power-of-two code)
// z_axis: the kernels bundle 8 adjacent z columns, so Nz must be a multiple of 8 (12 and 20 are x / y lengths only)
int next_supported_size(int n, bool pow2_only, bool z_axis) {
    if (pow2_only) return next_pow2_min8(n);
    static const int sizes[] = {8, 12, 16, 20, 24, 32, 40, 48, 64, 80, 96, 128, 160, 192, 256, 320, 384, 512, 768, 1024};
    for (int s : sizes)
        if (s >= n && !(z_axis && s % 8 != 0)) return s;
    return 1024;
}

// tables of k_dct1_warp<M> for this plan (built on first use, freed with the plan)
template <int M>
int dct_warp_tables(fsp_plan* p, double** lane, double2** roots) {
    for (size_t i = 0; i < p->dct_len.size(); ++i)
        if (p->dct_len[i] == M) { *lane = p->dct_lane[i]; *roots = p->dct_roots[i]; return FSP_OK; }
    double* l = nullptr;
    double2* r = nullptr;
    int rc = lane_table_for<M>(&l, &p->bytes);
    if (rc != FSP_OK) return rc;
    std::vector<double2> hst((size_t)M + 1);
    for (int m = 0; m <= M; ++m) hst[m] = unit_root(m, 2L * M);
    if ((rc = upload_table(&r, hst, &p->bytes)) != FSP_OK) { cudaFree(l); return rc; }
    p->dct_len.push_back(M); p->dct_lane.push_back(l); p->dct_roots.push_back(r);
    *lane = l; *roots = r;
    return FSP_OK;
}
template <int M>
int launch_dct1_warp(fsp_plan* p, const double* in, double* out, int nout, long nA, long nB, const long* ai, const long* ao,
                     double scale, const GLFill* fill) {
    using Cfg = Fft2Cfg<M>;
    constexpr int G = 32 / Cfg::T, WARPS = 8;
    double* lane = nullptr;
    double2* roots = nullptr;
    int rc = dct_warp_tables<M>(p, &lane, &roots);
    if (rc != FSP_OK) return rc;
    const size_t smem = sizeof(double2) * (size_t)(WARPS * G * Cfg::BUF);
    const long ngroups = (nA * nB + G - 1) / G;
    long grid = (ngroups + WARPS - 1) / WARPS;
    if (grid > (long)p->sm_count) grid = p->sm_count;
    if (fill) {
        { static OccCache optin; const int rc_ = cached_smem_optin(optin, p->device, k_dct1_warp<M, true>, smem); if (rc_ != FSP_OK) return rc_; }
        k_dct1_warp<M, true><<<(unsigned)grid, WARPS * 32, smem, p->stream>>>(in, out, nout, nA, nB, ai[0], ai[1], ai[2], ao[0], ao[1], ao[2],
                                                                          scale, *fill, lane, roots);
    } else {
        { static OccCache optin; const int rc_ = cached_smem_optin(optin, p->device, k_dct1_warp<M, false>, smem); if (rc_ != FSP_OK) return rc_; }
        k_dct1_warp<M, false><<<(unsigned)grid, WARPS * 32, smem, p->stream>>>(in, out, nout, nA, nB, ai[0], ai[1], ai[2], ao[0], ao[1], ao[2],
                                                                           scale, GLFill{0.0, 0.0, 0.0, 0.0, 0}, lane, roots);
    }
    CU(cudaGetLastError());
    return FSP_OK;
}

// batched DCT-I along one axis of a real 3-D array (C order), output pruned to nout along that axis.
// fill != nullptr (axis 2 only): the input array does not exist, its values are G_L evaluated inside the kernel.
template <int C>
int launch_dct1_tile(fsp_plan* p, const double* in, double* out, int n, int nout, long nA, long nB, const long* ai,
                     const long* ao, double scale, size_t smem, int threads, const GLFill* fill) {
    if (fill) {
        { static OccCache optin; const int rc_ = cached_smem_optin(optin, p->device, k_dct1_tile<C, true>, smem); if (rc_ != FSP_OK) return rc_; }
        k_dct1_tile<C, true><<<(unsigned)(nA * ((nB + C - 1) / C)), threads, smem, p->stream>>>(
            in, out, n, nout, nB, ai[0], ai[1], ai[2], ao[0], ao[1], ao[2], scale, *fill);
    } else {
        { static OccCache optin; const int rc_ = cached_smem_optin(optin, p->device, k_dct1_tile<C, false>, smem); if (rc_ != FSP_OK) return rc_; }
        k_dct1_tile<C, false><<<(unsigned)(nA * ((nB + C - 1) / C)), threads, smem, p->stream>>>(
            in, out, n, nout, nB, ai[0], ai[1], ai[2], ao[0], ao[1], ao[2], scale, GLFill{0.0, 0.0, 0.0, 0.0, 0});
    }
    CU(cudaGetLastError());
    return FSP_OK;
}
// DCT-I of an nA x nB grid of pencils with explicit strides: element k of pencil (a, b) at in[a ai[0] + b ai[1] + k ai[2]],
// output d at out[a ao[0] + b ao[1] + d ao[2]]; b is the dimension the kernels coalesce over.  kNoTileKernel when none of
// the pencil-grid kernels takes this length.
constexpr int kNoTileKernel = 1;
int dct1_strided(fsp_plan* p, const double* in, double* out, int n, int nout, long nA, long nB, const long ai[3],
                 const long ao[3], double scale, const GLFill* fill) {
    const int Lf = 2 * n;
    if ((n & (n - 1)) != 0) {   // not a power of two: the cosine sum as written (k_dct1_direct)
        constexpr int C = 8;
        const size_t smem = sizeof(double) * ((size_t)2 * n + (size_t)(n + 1) * C);
        if (smem > 200 * 1024) return FSP_ERR_INVALID_ARG;
        if (fill) {
            { static OccCache optin; const int rc_ = cached_smem_optin(optin, p->device, k_dct1_direct<C, true>, smem); if (rc_ != FSP_OK) return rc_; }
            k_dct1_direct<C, true><<<(unsigned)(nA * ((nB + C - 1) / C)), 256, smem, p->stream>>>(
                in, out, n, nout, nB, ai[0], ai[1], ai[2], ao[0], ao[1], ao[2], scale, *fill);
        } else {
            { static OccCache optin; const int rc_ = cached_smem_optin(optin, p->device, k_dct1_direct<C, false>, smem); if (rc_ != FSP_OK) return rc_; }
            k_dct1_direct<C, false><<<(unsigned)(nA * ((nB + C - 1) / C)), 256, smem, p->stream>>>(
                in, out, n, nout, nB, ai[0], ai[1], ai[2], ao[0], ao[1], ao[2], scale, GLFill{0.0, 0.0, 0.0, 0.0, 0});
        }
        CU(cudaGetLastError());
        return FSP_OK;
    }
    if (n >= 8 && n <= 1024) {   // the warp-level transform of the solve, one pencil per lane group (k_dct1_warp)
        switch (n) {
            case 8: return launch_dct1_warp<8>(p, in, out, nout, nA, nB, ai, ao, scale, fill);
            case 16: return launch_dct1_warp<16>(p, in, out, nout, nA, nB, ai, ao, scale, fill);
            case 32: return launch_dct1_warp<32>(p, in, out, nout, nA, nB, ai, ao, scale, fill);
            case 64: return launch_dct1_warp<64>(p, in, out, nout, nA, nB, ai, ao, scale, fill);
            case 128: return launch_dct1_warp<128>(p, in, out, nout, nA, nB, ai, ao, scale, fill);
            case 256: return launch_dct1_warp<256>(p, in, out, nout, nA, nB, ai, ao, scale, fill);
            case 512: return launch_dct1_warp<512>(p, in, out, nout, nA, nB, ai, ao, scale, fill);
            default: return launch_dct1_warp<1024>(p, in, out, nout, nA, nB, ai, ao, scale, fill);
        }
    }
    // Stockham tile kernel, C pencils per CTA.  Several CTAs per SM: the stages are latency-bound (one butterfly per
    // thread between two barriers)
    auto tile_smem = [&](int C) { return sizeof(double2) * ((size_t)n + (size_t)C * Lf); };
    if (tile_smem(8) <= 72 * 1024) return launch_dct1_tile<8>(p, in, out, n, nout, nA, nB, ai, ao, scale, tile_smem(8), 512, fill);
    if (tile_smem(4) <= 76 * 1024) return launch_dct1_tile<4>(p, in, out, n, nout, nA, nB, ai, ao, scale, tile_smem(4), 256, fill);
    if (tile_smem(2) <= 100 * 1024) return launch_dct1_tile<2>(p, in, out, n, nout, nA, nB, ai, ao, scale, tile_smem(2), 512, fill);
    if (tile_smem(4) <= 200 * 1024) return launch_dct1_tile<4>(p, in, out, n, nout, nA, nB, ai, ao, scale, tile_smem(4), 1024, fill);
    if (tile_smem(2) <= 200 * 1024) return launch_dct1_tile<2>(p, in, out, n, nout, nA, nB, ai, ao, scale, tile_smem(2), 512, fill);
    return kNoTileKernel;
}
// the same along one axis of a C-order array: pencils tiled along the contiguous dimension (z; y when the axis is z)
int dct1_axis(fsp_plan* p, const double* in, double* out, const long in_dims[3], const long out_dims[3],
              int axis, int n, int nout, double scale, const GLFill* fill = nullptr) {
    const long is[3] = {in_dims[1] * in_dims[2], in_dims[2], 1};
    const long os[3] = {out_dims[1] * out_dims[2], out_dims[2], 1};
    const int o1 = (axis + 1) % 3, o2 = (axis + 2) % 3;
    const long n1 = in_dims[o1], n2 = in_dims[o2];
    const int Lf = 2 * n;
    const int bdim = axis == 2 ? 1 : 2, adim = axis == 2 ? 0 : (axis == 0 ? 1 : 0);
    const long ai[3] = {is[adim], is[bdim], is[axis]}, ao[3] = {os[adim], os[bdim], os[axis]};
    const int rc = dct1_strided(p, in, out, n, nout, in_dims[adim], in_dims[bdim], ai, ao, scale, fill);
    if (rc != kNoTileKernel) return rc;
    if (fill) return FSP_ERR_INVALID_ARG;   // (lengths beyond the tile kernels: m_d N_d > 7264 is rejected before)
    const size_t smem = sizeof(double2) * 2 * (size_t)Lf;
    { static OccCache optin; const int rc_ = cached_smem_optin(optin, p->device, k_dct1_pencils, smem); if (rc_ != FSP_OK) return rc_; }
    int threads = Lf / 2 < 256 ? (Lf / 2 < 32 ? 32 : Lf / 2) : 256;
    k_dct1_pencils<<<(unsigned)(n1 * n2), threads, smem, p->stream>>>(in, out, n, nout, is[axis], os[axis], n2,
                                                                      is[o1], is[o2], os[o1], os[o2], scale);
    CU(cudaGetLastError());
    return FSP_OK;
}
// the y pass followed by the x pass of a 3-D DCT-I, src[a < na][b < nb][z < nz1] -> dst[Nx+1][Ny+1][nz1], through an
// intermediate `mid` stored [dy][a][z] -- dy OUTERMOST, so that the x pass reads pencils whose elements are nz1 doubles
// apart instead of (Ny+1) nz1 (2 MB at 512^3: one page per element).  y_only / x_only run one half (chunked callers).
int dct1_y_then_x(fsp_plan* p, const double* src, double* mid, double* dst, long na_total, long a0, long na, long nb_in,
                  long nz1, int ny, int nyout, int nx, int nxout, double scale, bool do_y, bool do_x) {
    int rc;
    if (do_y) {   // src[a][ky][z] (chunk of na planes starting at plane a0 of na_total) -> mid[dy][a0 + a][z]
        const long ai[3] = {nb_in * nz1, 1, nz1}, ao[3] = {nz1, 1, na_total * nz1};
        rc = dct1_strided(p, src, mid + (size_t)a0 * nz1, ny, nyout, na, nz1, ai, ao, 1.0, nullptr);
        if (rc != FSP_OK) return rc == kNoTileKernel ? FSP_ERR_INVALID_ARG : rc;
    }
    if (do_x) {   // mid[dy][kx][z] -> dst[dx][dy][z]
        const long ai[3] = {na_total * nz1, 1, nz1}, ao[3] = {nz1, 1, (long)nyout * nz1};
        rc = dct1_strided(p, mid, dst, nx, nxout, nyout, nz1, ai, ao, scale, nullptr);
        if (rc != FSP_OK) return rc == kNoTileKernel ? FSP_ERR_INVALID_ARG : rc;
    }
    return FSP_OK;
}

// tile geometry shared by the plain-VG passes: C pencils adjacent along the contiguous dimension (z; y when the
// transform axis is z), nA x nB pencil grid, strides {sA, sB, sK} of a C-order array with dimensions dims
struct AxisTiling { long nA, nB, sA, sB, sK; };
AxisTiling axis_tiling(const long dims[3], int axis) {
    const long st[3] = {dims[1] * dims[2], dims[2], 1};
    const int bdim = axis == 2 ? 1 : 2, adim = axis == 2 ? 0 : (axis == 0 ? 1 : 0);
    return AxisTiling{dims[adim], dims[bdim], st[adim], st[bdim], st[axis]};
}

template <int C>
int launch_ifft_tile(fsp_plan* p, double2* data, int Lf, long nA, long nB, long sA, long sB, long sK, size_t smem) {
    { static OccCache optin; const int rc_ = cached_smem_optin(optin, p->device, k_ifft_tile<C>, smem); if (rc_ != FSP_OK) return rc_; }
    k_ifft_tile<C><<<(unsigned)(nA * ((nB + C - 1) / C)), smem <= 72 * 1024 ? 512 : 1024, smem, p->stream>>>(data, Lf, nB, sA, sB, sK);
    CU(cudaGetLastError());
    return FSP_OK;
}
// in-place unscaled inverse DFT along `axis` of the complex array data[dims], for the pencils whose index along the
// tiled dimension is below nB_used
int ifft_axis(fsp_plan* p, double2* data, const long dims[3], int axis, long nA_used, long nB_used) {
    const AxisTiling t = axis_tiling(dims, axis);
    const int Lf = (int)dims[axis];
    auto smem = [&](int C) { return sizeof(double2) * ((size_t)Lf / 2 + 2 * (size_t)C * Lf); };
    const size_t cap = 200 * 1024;
    if (smem(8) <= 72 * 1024) return launch_ifft_tile<8>(p, data, Lf, nA_used, nB_used, t.sA, t.sB, t.sK, smem(8));
    if (smem(4) <= cap) return launch_ifft_tile<4>(p, data, Lf, nA_used, nB_used, t.sA, t.sB, t.sK, smem(4));
    if (smem(2) <= cap) return launch_ifft_tile<2>(p, data, Lf, nA_used, nB_used, t.sA, t.sB, t.sK, smem(2));
    if (smem(1) <= cap) return launch_ifft_tile<1>(p, data, Lf, nA_used, nB_used, t.sA, t.sB, t.sK, smem(1));
    return FSP_ERR_INVALID_ARG;
}
template <int C>
int launch_c2r_tile(fsp_plan* p, const double2* in, double* out, int Lf, int nout, long nA, long nB, const AxisTiling& ti,
                    const AxisTiling& to, double scale, size_t smem) {
    { static OccCache optin; const int rc_ = cached_smem_optin(optin, p->device, k_c2r_tile<C>, smem); if (rc_ != FSP_OK) return rc_; }
    k_c2r_tile<C><<<(unsigned)(nA * ((nB + C - 1) / C)), smem <= 72 * 1024 ? 512 : 1024, smem, p->stream>>>(
        in, out, Lf, nout, nB, ti.sA, ti.sB, ti.sK, to.sA, to.sB, to.sK, scale);
    CU(cudaGetLastError());
    return FSP_OK;
}
// C2R along `axis` (half spectrum Lf/2 + 1 in, nout reals out), pencils (a < nA_used, b < nB_used)
int c2r_axis(fsp_plan* p, const double2* in, double* out, const long in_dims[3], const long out_dims[3], int axis, int Lf,
             int nout, long nA_used, long nB_used, double scale) {
    const AxisTiling ti = axis_tiling(in_dims, axis), to = axis_tiling(out_dims, axis);
    auto smem = [&](int C) { return sizeof(double2) * ((size_t)Lf / 2 + (size_t)C * Lf); };
    const size_t cap = 200 * 1024;
    if (smem(8) <= 72 * 1024) return launch_c2r_tile<8>(p, in, out, Lf, nout, nA_used, nB_used, ti, to, scale, smem(8));
    if (smem(4) <= cap) return launch_c2r_tile<4>(p, in, out, Lf, nout, nA_used, nB_used, ti, to, scale, smem(4));
    if (smem(2) <= cap) return launch_c2r_tile<2>(p, in, out, Lf, nout, nA_used, nB_used, ti, to, scale, smem(2));
    return FSP_ERR_INVALID_ARG;
}

struct ScopedFree {
    std::vector<void*> ptrs;
    ~ScopedFree() {
        for (void* q : ptrs)
            if (q) cudaFree(q);
    }
};

int precompute_impl(fsp_plan* p) {
    const int Nx = p->Nx, Ny = p->Ny, Nz = p->Nz;
    const double hx = p->h[0], hy = p->h[1], hz = p->h[2];
    const long tdims[3] = {Nx + 1, Ny + 1, Nz + 1};
    const long tcount = tdims[0] * tdims[1] * tdims[2];
    ScopedFree tmp;
    size_t peak = 0;
    const int blk = 256;
    struct TransientTables {   // sharded plan, y-z stage: T and Goct live for the duration of this call only
        fsp_plan* p; bool on;
        ~TransientTables() { if (on) { cudaFree(p->T); cudaFree(p->Goct); p->T = nullptr; p->Goct = nullptr; } }
    } transient{p, false};
    if (p->stage == 2) {
        int rc = dev_alloc(&p->T, (size_t)tcount, &peak);
        if (rc == FSP_OK) rc = dev_alloc(&p->Goct, (size_t)tcount, &peak);
        transient.on = true;
        if (rc != FSP_OK) return rc;
    }

    if (p->algorithm == FSP_HOCKNEY) {
        k_fill_he<<<grid_for(tcount, blk), blk, 0, p->stream>>>(p->T, Nx, Ny, Nz, hx, hy, hz, p->g0);
        CU(cudaGetLastError());
        if (p->periodic) {   // (set_param has checked: FSP_HOCKNEY, mesh not embedded)
            k_fold_periodic<<<grid_for(tcount, blk), blk, 0, p->stream>>>(p->T, Nx, Ny, Nz, p->periodic);
            CU(cudaGetLastError());
        }
    } else {
        const double Lx = Nx * hx, Ly = Ny * hy, Lz = Nz * hz;
        const double L = p->alpha * std::sqrt(Lx * Lx + Ly * Ly + Lz * Lz);
        const double scale = 1.0 / ((4.0 * Nx * hx) * (4.0 * Ny * hy) * (4.0 * Nz * hz));
        if (p->algorithm == FSP_VICO) {
            // (4N)^3 lattice of G_L, real, stored as its C2R half spectrum (2Nx+1) x 4Ny x 4Nz complex: fill, unscaled
            // inverse DFT along z (all pencils), along y (columns dz <= Nz only), C2R along x for dy <= Ny, dz <= Nz
            // straight into T (the restriction of PAPER.md:98)
            const long gd[3] = {2L * Nx + 1, 4L * Ny, 4L * Nz};
            const size_t gcount = (size_t)gd[0] * gd[1] * gd[2];
            double2* g = nullptr;
            int rc = dev_alloc(&g, gcount, &peak);
            if (rc != FSP_OK) return rc;
            tmp.ptrs.push_back(g);
            k_fill_gl_vg_half<<<grid_for((long)gcount, blk), blk, 0, p->stream>>>(g, Nx, Ny, Nz, hx, hy, hz, L);
            CU(cudaGetLastError());
            if ((rc = ifft_axis(p, g, gd, 2, gd[0], gd[1])) != FSP_OK) return rc;
            if ((rc = ifft_axis(p, g, gd, 1, gd[0], Nz + 1)) != FSP_OK) return rc;
            if ((rc = c2r_axis(p, g, p->T, gd, tdims, 0, 4 * Nx, Nx + 1, Ny + 1, Nz + 1, scale)) != FSP_OK) return rc;
        } else {
            // (m_d N_d / 2 + 1) real grid per axis, DCT-I per axis with output pruned to N_d + 1
            // (PAPER.md:100-102 with m = 4; FSP_VICO_SAFE: m_d = 4, doubled while m_d < 1 + L / L_d, R17)
            int m[3] = {4, 4, 4};
            if (p->algorithm == FSP_VICO_SAFE) {
                const double Ld[3] = {Lx, Ly, Lz};
                for (int d = 0; d < 3; ++d)
                    while ((double)m[d] < 1.0 + L / Ld[d]) m[d] *= 2;
            }
            p->vg_m[0] = m[0]; p->vg_m[1] = m[1]; p->vg_m[2] = m[2];
            const int nx = m[0] * Nx / 2, ny = m[1] * Ny / 2, nz = m[2] * Nz / 2;   // DCT-I sizes are n + 1
            // the DCT kernel holds two arrays of 2n complex values in shared memory
            if (sizeof(double2) * 4 * (size_t)(nx > ny ? (nx > nz ? nx : nz) : (ny > nz ? ny : nz)) > 227 * 1024)
                return FSP_ERR_INVALID_ARG;
            const double vscale = 1.0 / (((double)m[0] * Nx * hx) * ((double)m[1] * Ny * hy) * ((double)m[2] * Nz * hz));
            // The lattice f[kx][ky][kz] is never stored: the z pass evaluates G_L itself (k_dct1_tile<., FILL>).  It runs
            // a chunk of kx planes at a time through a[kx][ky][dz] (in the plan's workspace B1), the y pass takes the
            // chunk to b[kx][dy][dz] (workspace B2), the x pass b -> T.  No transient memory when the workspace holds
            // a plane of a and the whole of b (always for the paper's m = 4), else it is allocated.
            const long Kx = nx + 1L, Ky = ny + 1L;
            if ((nz & (nz - 1)) == 0 && sizeof(double2) * 5 * (size_t)nz > 200 * 1024) {
                // the z transform is too long for the tile kernels (m_z N_z > 5120): the unfused route, lattice in memory
                const long fd[3] = {nx + 1L, ny + 1L, nz + 1L};
                const long ad[3] = {fd[0], fd[1], Nz + 1};
                const long bd[3] = {fd[0], Ny + 1, Nz + 1};
                double *f = nullptr, *a = nullptr, *b = nullptr;
                int rc = dev_alloc(&f, (size_t)fd[0] * fd[1] * fd[2], &peak);
                if (rc != FSP_OK) return rc;
                tmp.ptrs.push_back(f);
                if ((rc = dev_alloc(&a, (size_t)ad[0] * ad[1] * ad[2], &peak)) != FSP_OK) return rc;
                tmp.ptrs.push_back(a);
                if ((rc = dev_alloc(&b, (size_t)bd[0] * bd[1] * bd[2], &peak)) != FSP_OK) return rc;
                tmp.ptrs.push_back(b);
                k_fill_gl_vg2<<<grid_for(fd[0] * fd[1] * fd[2], blk), blk, 0, p->stream>>>(f, Nx, Ny, Nz, hx, hy, hz, L, m[0], m[1], m[2]);
                CU(cudaGetLastError());
                if ((rc = dct1_axis(p, f, a, fd, ad, 2, nz, Nz + 1, 1.0)) != FSP_OK) return rc;
                if ((rc = dct1_axis(p, a, b, ad, bd, 1, ny, Ny + 1, 1.0)) != FSP_OK) return rc;
                if ((rc = dct1_axis(p, b, p->T, bd, tdims, 0, nx, Nx + 1, vscale)) != FSP_OK) return rc;
            } else {
            const size_t plane_a = (size_t)Ky * (Nz + 1), count_b = (size_t)Kx * (Ny + 1) * (Nz + 1);
            const size_t cap1 = p->b1_count * 2, cap2 = p->b2_count * 2;   // doubles in B1, B2
            double *a = reinterpret_cast<double*>(p->B1), *b = reinterpret_cast<double*>(p->B2);
            long chunk = (long)(cap1 / plane_a);
            int rc;
            if (chunk < 1) {
                chunk = Kx < 64 ? Kx : 64;
                if ((rc = dev_alloc(&a, (size_t)chunk * plane_a, &peak)) != FSP_OK) return rc;
                tmp.ptrs.push_back(a);
            }
            if (chunk > Kx) chunk = Kx;
            if (count_b > cap2) {
                if ((rc = dev_alloc(&b, count_b, &peak)) != FSP_OK) return rc;
                tmp.ptrs.push_back(b);
            }
            const double PI2 = 6.28318530717958647692;
            for (long a0 = 0; a0 < Kx; a0 += chunk) {
                const long nc = Kx - a0 < chunk ? Kx - a0 : chunk;
                const long fd[3] = {nc, Ky, nz + 1L};
                const long ad[3] = {nc, Ky, Nz + 1};
                const GLFill gl{PI2 / ((double)m[0] * Nx * hx), PI2 / ((double)m[1] * Ny * hy), PI2 / ((double)m[2] * Nz * hz), L, a0};
                if ((rc = dct1_axis(p, nullptr, a, fd, ad, 2, nz, Nz + 1, 1.0, &gl)) != FSP_OK) return rc;
                if ((rc = dct1_y_then_x(p, a, b, nullptr, Kx, a0, nc, Ky, Nz + 1, ny, Ny + 1, nx, Nx + 1, 1.0, true, false)) != FSP_OK) return rc;
            }
            if ((rc = dct1_y_then_x(p, nullptr, b, p->T, Kx, 0, Kx, Ky, Nz + 1, ny, Ny + 1, nx, Nx + 1, vscale, false, true)) != FSP_OK) return rc;
            }
        }
    }
    // Ghat octant = 3-D DCT-I of T (size N_d + 1 per axis)
    {
        double* u = reinterpret_cast<double*>(p->B1);   // the solve's workspace serves as scratch when it is big enough
        int rc = FSP_OK;
        if ((size_t)tcount > p->b1_count * 2) {
            if ((rc = dev_alloc(&u, (size_t)tcount, &peak)) != FSP_OK) return rc;
            tmp.ptrs.push_back(u);
        }
        if ((rc = dct1_axis(p, p->T, p->Goct, tdims, tdims, 2, Nz, Nz + 1, 1.0)) != FSP_OK) return rc;
        if ((rc = dct1_y_then_x(p, p->Goct, u, p->Goct, Nx + 1, 0, Nx + 1, Ny + 1, Nz + 1, Ny, Ny + 1, Nx, Nx + 1, 1.0, true, true)) != FSP_OK) return rc;
    }
    // scale: hx hy hz / (8 Nx Ny Nz) (inverse DFT) / 2 (K1 produces 2X)
    const double gscale = hx * hy * hz / (8.0 * (double)Nx * (double)Ny * (double)Nz) * 0.5;
    {
        // (a sharded plan keeps the rows of its own kx planes only)
        const long gk_total = (long)p->planes * (Ny + 1) * (Nz + 2);
        const double* goct = p->Goct + (size_t)p->kx0 * (Ny + 1) * (Nz + 1);
        p->gk_pfa = z_uses_pf(Nz) && p->k3_variant == 0;
        p->gk_natural = !p->gk_pfa && ((Nz == 256 || Nz == 512) ? p->k3_variant == 0 : (z_uses_g2(Nz) && p->k3_variant != 1));
        if (p->gk_pfa) {
            const int B = pf_radix(Nz), P = 2 * Nz / B;
            const int c1 = P * mod_inverse(P % B, B), c2 = B * mod_inverse(B % P, P);   // k = (c1 k1 + c2 k2) mod 2 Nz
            const long tot = (long)p->planes * (Ny + 1) * 2 * Nz;
            k_layout_spectrum_pfa<<<grid_for(tot, blk), blk, 0, p->stream>>>(goct, p->Gk, p->planes - 1, Ny, Nz, P, c1, c2, gscale);
        } else if (p->gk_natural) k_layout_spectrum_nat<<<grid_for(gk_total, blk), blk, 0, p->stream>>>(goct, p->Gk, p->planes - 1, Ny, Nz, gscale);
        else k_layout_spectrum_oct<<<grid_for(gk_total, blk), blk, 0, p->stream>>>(goct, p->Gk, p->planes - 1, Ny, Nz, gscale);
    }
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(p->stream));
    p->peak_transient = peak;
    return FSP_OK;
}

void free_plan_memory(fsp_plan* p) {
    for (double* q : p->dct_lane) cudaFree(q);
    for (double2* q : p->dct_roots) cudaFree(q);
    p->dct_lane.clear(); p->dct_roots.clear(); p->dct_len.clear();
    cudaFree(p->B1); cudaFree(p->B2); cudaFree(p->B3); cudaFree(p->rho_pad); cudaFree(p->phi_pad); cudaFree(p->E_stage); cudaFree(p->rho_stage2); cudaFree(p->phi_stage2); cudaFree(p->Gk); cudaFree(p->LTz); cudaFree(p->LTzs); cudaFree(p->LTzf); cudaFree(p->LTy); cudaFree(p->LTyf); cudaFree(p->LTx); cudaFree(p->T); cudaFree(p->Goct);
    cudaFree(p->Wx); cudaFree(p->Wy); cudaFree(p->Wz); cudaFree(p->rho_stage); cudaFree(p->phi_stage);
    for (cudaEvent_t e : p->events) cudaEventDestroy(e);
    p->events.clear();
    for (int i = 0; i < 2; ++i) {
        if (p->ev_h2d[i]) cudaEventDestroy(p->ev_h2d[i]);
        if (p->ev_solve[i]) cudaEventDestroy(p->ev_solve[i]);
        if (p->ev_d2h[i]) cudaEventDestroy(p->ev_d2h[i]);
    }
    if (p->s_h2d) cudaStreamDestroy(p->s_h2d);
    if (p->s_d2h) cudaStreamDestroy(p->s_d2h);
}

}  // namespace

extern "C" {

int fsp_version(void) { return FSP_VERSION_NUM; }

const char* fsp_strerror(int code) {
    switch (code) {
        case FSP_OK: return "success";
        case FSP_ERR_INVALID_ARG: return "invalid argument";
        case FSP_ERR_NOT_PRECOMPUTED: return "fsp_precompute_green has not been called";
        case FSP_ERR_OUT_OF_MEMORY: return "device memory allocation failed";
        case FSP_ERR_CUDA: return "CUDA runtime or kernel launch error";
        case FSP_ERR_NO_DEVICE: return "no usable CUDA device";
        case FSP_ERR_STATIC_CAPACITY: return "table larger than the static scratch array (FSP_STATIC_MAX_DOUBLES)";
        default: return "unknown error code";
    }
}

const char* fsp_kernel_name(int i) {
    static const char* names[FSP_NUM_SOLVE_KERNELS] = {"k_fwd_x_r2c", "k_fwd_y", "k_conv_z", "k_inv_y", "k_inv_x_c2r"};
    return (i >= 0 && i < FSP_NUM_SOLVE_KERNELS) ? names[i] : "";
}

// stage / kx0 / planes: see fsp_plan.  Stages 1 and 2 are the two halves of a sharded plan (power-of-two meshes only).
static int plan_create_impl(fsp_plan** out, int Nx, int Ny, int Nz, const double* h, int algorithm, void* cuda_stream,
                            int stage, int kx0, int planes_req) {
    if (!out) return FSP_ERR_INVALID_ARG;
    *out = nullptr;
    if (!h || !(h[0] > 0.0) || !(h[1] > 0.0) || !(h[2] > 0.0)) return FSP_ERR_INVALID_ARG;
    if (!std::isfinite(h[0]) || !std::isfinite(h[1]) || !std::isfinite(h[2])) return FSP_ERR_INVALID_ARG;
    if (Nx < 2 || Ny < 2 || Nz < 2 || Nx > 1024 || Ny > 1024 || Nz > 1024) return FSP_ERR_INVALID_ARG;
    const int Ux = Nx, Uy = Ny, Uz = Nz;
    // transform lengths are 2^k, 3 * 2^k or 5 * 2^k: any other mesh is embedded in the next such mesh (R19)
    Nx = next_supported_size(Ux, algorithm == FSP_VICO, false); Ny = next_supported_size(Uy, algorithm == FSP_VICO, false);
    Nz = next_supported_size(Uz, algorithm == FSP_VICO, true);
    if (algorithm != FSP_HOCKNEY && algorithm != FSP_VICO && algorithm != FSP_VICO_2 && algorithm != FSP_VICO_SAFE) return FSP_ERR_INVALID_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        (void)cudaGetLastError();
        return FSP_ERR_NO_DEVICE;
    }
    fsp_plan* p = new (std::nothrow) fsp_plan();
    if (!p) return FSP_ERR_OUT_OF_MEMORY;
    p->Nx = Nx; p->Ny = Ny; p->Nz = Nz;
    p->Ux = Ux; p->Uy = Uy; p->Uz = Uz;
    p->padded = Ux != Nx || Uy != Ny || Uz != Nz;
    p->h[0] = h[0]; p->h[1] = h[1]; p->h[2] = h[2];
    p->algorithm = algorithm;
    p->stream = static_cast<cudaStream_t>(cuda_stream);
    p->g0 = 1.0 / (4.0 * 3.14159265358979323846);
    p->alpha = 1.1;
    int rc = FSP_OK;
    cudaDeviceProp prop{};
    if (cudaGetDevice(&p->device) != cudaSuccess || cudaGetDeviceProperties(&prop, p->device) != cudaSuccess) rc = FSP_ERR_NO_DEVICE;
    if (rc == FSP_OK && prop.major != 10) rc = FSP_ERR_NO_DEVICE;  // the library holds sm_100a code only
    if (rc == FSP_OK && (p->device < 0 || p->device >= kMaxDevices)) rc = FSP_ERR_NO_DEVICE;
    if (stage != 0 && p->padded) rc = FSP_ERR_INVALID_ARG;
    const int planes = stage == 2 ? planes_req : Nx + 1;
    p->stage = stage; p->planes = planes; p->kx0 = stage == 2 ? kx0 : 0;
    const bool want_x = stage != 2, want_yz = stage != 1;
    const size_t n1 = (size_t)planes * Ny * Nz, n2 = (size_t)planes * 2 * Ny * Nz;
    const size_t nt = (size_t)(Nx + 1) * (Ny + 1) * (Nz + 1);
    p->b1_count = n1; p->b2_count = want_yz ? n2 : 0;
    if (rc == FSP_OK && p->padded) rc = dev_alloc(&p->rho_pad, (size_t)Nx * Ny * Nz, &p->bytes);
    if (rc == FSP_OK && p->padded) rc = dev_alloc(&p->phi_pad, (size_t)Nx * Ny * Nz, &p->bytes);
    if (rc == FSP_OK && p->padded && cudaMemset(p->rho_pad, 0, sizeof(double) * (size_t)Nx * Ny * Nz) != cudaSuccess) rc = FSP_ERR_CUDA;
    if (rc == FSP_OK) rc = dev_alloc(&p->B1, n1, &p->bytes);
    if (rc == FSP_OK && want_yz) rc = dev_alloc(&p->B2, n2, &p->bytes);
    p->sm_count = prop.multiProcessorCount > 0 ? prop.multiProcessorCount : 148;
    if (rc == FSP_OK && want_yz) rc = dev_alloc(&p->Gk, (size_t)planes * (Ny + 1) * gk_row(Nz), &p->bytes);
    if (rc == FSP_OK && want_yz && z_uses_pf(Nz)) {   // stage-2 constants of the P-point sub-transforms, P = 2 Nz / B
        switch (2 * Nz / pf_radix(Nz)) {
            case 256: rc = lane_table_for<256>(&p->LTzf, &p->bytes); break;
            case 128: rc = lane_table_for<128>(&p->LTzf, &p->bytes); break;
            case 64: rc = lane_table_for<64>(&p->LTzf, &p->bytes); break;
            case 32: rc = lane_table_for<32>(&p->LTzf, &p->bytes); break;
            default: rc = lane_table_for<16>(&p->LTzf, &p->bytes); break;
        }
    }
    if (rc == FSP_OK && want_yz) rc = make_z_lane_table(p);
    if (rc == FSP_OK && want_yz && Nz == 512) rc = make_lane_table_512s(&p->LTzs, &p->bytes);
    if (rc == FSP_OK && want_yz && Nz == 512) rc = lane_table_for<1024>(&p->LTzf, &p->bytes);
    if (rc == FSP_OK && want_yz && Nz == 256) rc = lane_table_for<512>(&p->LTzf, &p->bytes);
    p->tile_x = want_x && (Nx == 128 || Nx == 256 || Nx == 512 || Nx == 1024) && ((long)Ny * Nz) % kC == 0;
    if (rc == FSP_OK && p->tile_x) rc = make_x_lane_table(p);
    if (rc == FSP_OK && p->tile_x) {
        const cuuint64_t plane = (cuuint64_t)Ny * Nz;
        const cuuint64_t dims[3] = {2 * plane, 2, (cuuint64_t)(Nx / 2)};
        const cuuint64_t strides[2] = {plane * 16, 2 * plane * 16};
        const cuuint32_t box[3] = {2 * (cuuint32_t)(Nx == 1024 ? 8 : kC), 1, (cuuint32_t)(Nx / 2 < 256 ? Nx / 2 : 256)};   // TileXI<M>::KC columns
        rc = make_tensor_map(&p->tmB1x, p->B1, 3, dims, strides, box);
    }
    p->tile_y = want_yz && (Ny == 128 || Ny == 256 || Ny == 512 || Ny == 1024) && Nz >= kW;
    const cuuint32_t kwy = Ny == 1024 ? 4 : kW;   // TileY<M>::KW: columns per tile of the y tile kernels
    if (rc == FSP_OK && p->tile_y) rc = make_y_lane_table(p);
    if (rc == FSP_OK && p->tile_y && Ny == 512) rc = lane_table_for<1024>(&p->LTyf, &p->bytes);
    if (rc == FSP_OK && p->tile_y) {
        const cuuint64_t dims[3] = {(cuuint64_t)2 * Nz, (cuuint64_t)Ny, (cuuint64_t)planes};
        const cuuint64_t strides[2] = {(cuuint64_t)Nz * 16, (cuuint64_t)Ny * Nz * 16};
        const cuuint32_t box[3] = {2 * kwy, (cuuint32_t)(Ny < 256 ? Ny : 256), 1};
        rc = make_tensor_map(&p->tmB1y, p->B1, 3, dims, strides, box);
    }
    if (rc == FSP_OK && p->tile_y) {
        const cuuint64_t dims[4] = {(cuuint64_t)2 * Nz, 2, (cuuint64_t)Ny, (cuuint64_t)planes};
        const cuuint64_t strides[3] = {(cuuint64_t)Nz * 16, (cuuint64_t)2 * Nz * 16, (cuuint64_t)2 * Ny * Nz * 16};
        const cuuint32_t box[4] = {2 * kwy, 1, (cuuint32_t)(Ny < 256 ? Ny : 256), 1};
        rc = make_tensor_map(&p->tmB2y, p->B2, 4, dims, strides, box);
    }
    // (the y-z stage of a sharded plan holds the table and the un-normalised octant only while its precompute runs)
    if (rc == FSP_OK && want_yz && stage == 0) rc = dev_alloc(&p->T, nt, &p->bytes);
    if (rc == FSP_OK && want_yz && stage == 0) rc = dev_alloc(&p->Goct, nt, &p->bytes);
    if (rc == FSP_OK && want_x) rc = make_table(&p->Wx, 2 * Nx, &p->bytes);
    if (rc == FSP_OK && want_yz) rc = make_table(&p->Wy, 2 * Ny, &p->bytes);
    if (rc == FSP_OK && want_yz) rc = make_table(&p->Wz, 2 * Nz, &p->bytes);
    if (rc != FSP_OK) {
        free_plan_memory(p);
        delete p;
        return rc;
    }
    *out = p;
    return FSP_OK;
}

int fsp_plan_create(fsp_plan** out, int Nx, int Ny, int Nz, const double* h, int algorithm, void* cuda_stream) {
    return plan_create_impl(out, Nx, Ny, Nz, h, algorithm, cuda_stream, 0, 0, 0);
}

int fsp_plan_set_param(fsp_plan* p, int which, double value) {
    if (!p || !std::isfinite(value)) return FSP_ERR_INVALID_ARG;
    if (which == FSP_PARAM_G0) { p->g0 = value; return FSP_OK; }
    if (which == FSP_PARAM_CHUNK_PLANES) {
        if (value < 0.0 || value > 4096.0) return FSP_ERR_INVALID_ARG;
        p->chunk_planes = (int)value;
        return FSP_OK;
    }
    if (which == FSP_PARAM_K2_VARIANT) {
        if (value != 0.0 && value != 1.0) return FSP_ERR_INVALID_ARG;
        p->k2_variant = (int)value;
        return FSP_OK;
    }
    if (which == FSP_PARAM_PERIODIC_FAST_Z) {
        if (value != 0.0 && value != 1.0) return FSP_ERR_INVALID_ARG;
        p->periodic_fast_z = value != 0.0;
        return FSP_OK;
    }
    if (which == FSP_PARAM_PERIODIC) {
        const int mask = (int)value;
        if (value != (double)mask || mask < 0 || mask > 7) return FSP_ERR_INVALID_ARG;
        // the nearest-image kernel is defined for the 1/r table; the period must be the caller's N_d, so no embedding
        if (mask != 0 && (p->algorithm != FSP_HOCKNEY || p->padded)) return FSP_ERR_INVALID_ARG;
        p->periodic = mask;
        p->precomputed = false;
        return FSP_OK;
    }
    if (which == FSP_PARAM_K3_VARIANT) {
        if (value != 0.0 && value != 1.0 && value != 2.0) return FSP_ERR_INVALID_ARG;
        p->k3_variant = (int)value;
        p->precomputed = false;   // the layout of the spectrum rows depends on the kernel
        return FSP_OK;
    }
    if (which == FSP_PARAM_ALPHA) {
        if (!(value > 1.0)) return FSP_ERR_INVALID_ARG;   // the window must exceed the domain diagonal
        p->alpha = value;
        return FSP_OK;
    }
    return FSP_ERR_INVALID_ARG;
}

int fsp_plan_set_spacing(fsp_plan* p, const double* h) {
    if (!p || !h) return FSP_ERR_INVALID_ARG;
    for (int d = 0; d < 3; ++d)
        if (!(h[d] > 0.0) || !std::isfinite(h[d])) return FSP_ERR_INVALID_ARG;
    p->h[0] = h[0]; p->h[1] = h[1]; p->h[2] = h[2];
    p->precomputed = false;   // the table and the spectrum belong to the old spacing
    return FSP_OK;
}

int fsp_precompute_green(fsp_plan* p) {
    if (!p || p->stage == 1) return FSP_ERR_INVALID_ARG;
    DeviceGuard dev_guard(p->device);
    p->precomputed = false;
    int rc = precompute_impl(p);
    if (rc != FSP_OK) {
        cudaStreamSynchronize(p->stream);
        (void)cudaGetLastError();
        return rc;
    }
    p->precomputed = true;
    return FSP_OK;
}

int fsp_solve(fsp_plan* p, const double* rho_dev, double* phi_dev) {
    if (!p || !rho_dev || !phi_dev || rho_dev == phi_dev) return FSP_ERR_INVALID_ARG;
    if (p->stage != 0) return FSP_ERR_INVALID_ARG;
    if (!p->precomputed) return FSP_ERR_NOT_PRECOMPUTED;
    DeviceGuard dev_guard(p->device);
    double* phi_user = nullptr;
    if (p->padded) {   // embed, solve on the transform mesh, crop
        int rce = embed_rho(p, rho_dev);
        if (rce != FSP_OK) return rce;
        rho_dev = p->rho_pad;
        phi_user = phi_dev;
        phi_dev = p->phi_pad;
    }
    cudaEvent_t* ev = nullptr;
    if (p->profiling) {
        if (p->events_used + 6 > p->events.size()) {
            for (int i = 0; i < 6; ++i) {
                cudaEvent_t e;
                CU(cudaEventCreate(&e));
                p->events.push_back(e);
            }
        }
        ev = &p->events[p->events_used];
        p->events_used += 6;
        CU(cudaEventRecord(ev[0], p->stream));
    }
    int rc;
    if ((rc = do_fwd_x(p, rho_dev)) != FSP_OK) return rc;
    if (ev) CU(cudaEventRecord(ev[1], p->stream));
    const int planes = p->Nx + 1;
    if (p->chunk_planes > 0 && p->chunk_planes < planes) {
        // plane-chunked middle: K2 -> K3 -> K4 on chunk_planes kx-planes at a time through the head of
        // B2, so that B2 stays resident in L2 between the three passes
        const size_t plane1 = (size_t)p->Ny * p->Nz;
        for (int kx0 = 0; kx0 < planes; kx0 += p->chunk_planes) {
            const int np = planes - kx0 < p->chunk_planes ? planes - kx0 : p->chunk_planes;
            if ((rc = do_fwd_y(p, kx0, p->B2, np)) != FSP_OK) return rc;
            if ((rc = do_conv_z(p, p->B2, kx0, np)) != FSP_OK) return rc;
            if ((rc = do_inv_y(p, p->B2, p->B1 + kx0 * plane1, np)) != FSP_OK) return rc;
        }
        if (ev) { CU(cudaEventRecord(ev[2], p->stream)); CU(cudaEventRecord(ev[3], p->stream)); CU(cudaEventRecord(ev[4], p->stream)); }
    } else {
    if ((rc = do_fwd_y(p, 0, p->B2, planes)) != FSP_OK) return rc;
    if (ev) CU(cudaEventRecord(ev[2], p->stream));
    if ((rc = do_conv_z(p, p->B2, 0, planes)) != FSP_OK) return rc;
    if (ev) CU(cudaEventRecord(ev[3], p->stream));
    if ((rc = do_inv_y(p, p->B2, p->B1, planes)) != FSP_OK) return rc;
    if (ev) CU(cudaEventRecord(ev[4], p->stream));
    }
    if ((rc = do_inv_x(p, phi_dev)) != FSP_OK) return rc;
    if (phi_user && (rc = crop_out(p, phi_user)) != FSP_OK) return rc;
    if (ev) CU(cudaEventRecord(ev[5], p->stream));
    CU(cudaGetLastError());
    return FSP_OK;
}

int fsp_solve_host(fsp_plan* p, const double* rho_host, double* phi_host) {
    if (!p || !rho_host || !phi_host) return FSP_ERR_INVALID_ARG;
    if (!p->precomputed) return FSP_ERR_NOT_PRECOMPUTED;
    DeviceGuard dev_guard(p->device);
    const size_t v = user_volume(p);
    if (!p->rho_stage) {
        int rc = dev_alloc(&p->rho_stage, v, &p->bytes);
        if (rc != FSP_OK) return rc;
        rc = dev_alloc(&p->phi_stage, v, &p->bytes);
        if (rc != FSP_OK) return rc;
    }
    CU(cudaMemcpyAsync(p->rho_stage, rho_host, v * sizeof(double), cudaMemcpyHostToDevice, p->stream));
    int rc = fsp_solve(p, p->rho_stage, p->phi_stage);
    if (rc != FSP_OK) return rc;
    CU(cudaMemcpyAsync(phi_host, p->phi_stage, v * sizeof(double), cudaMemcpyDeviceToHost, p->stream));
    CU(cudaStreamSynchronize(p->stream));
    return FSP_OK;
}

// the pipeline of fsp_solve_host_batch (the caller drains the three streams if this returns an error)
static int batch_pipeline(fsp_plan* p, int n, const double* const* rho_hosts, double* const* phi_hosts, size_t v) {
    int rc;
    double* rs[2] = {p->rho_stage, p->rho_stage2};
    double* ps[2] = {p->phi_stage, p->phi_stage2};
    // earlier work on the plan's stream may still use the staging buffers
    CU(cudaEventRecord(p->ev_solve[0], p->stream));
    CU(cudaStreamWaitEvent(p->s_h2d, p->ev_solve[0], 0));
    CU(cudaStreamWaitEvent(p->s_d2h, p->ev_solve[0], 0));
    for (int i = 0; i < n; ++i) {
        const int s = i & 1;
        // copy-in of solve i: its staging buffer is free once solve i-2 has run
        if (i >= 2) CU(cudaStreamWaitEvent(p->s_h2d, p->ev_solve[s], 0));
        CU(cudaMemcpyAsync(rs[s], rho_hosts[i], v * sizeof(double), cudaMemcpyHostToDevice, p->s_h2d));
        CU(cudaEventRecord(p->ev_h2d[s], p->s_h2d));
        // solve i: needs its input, and its output buffer back from the copy-out of solve i-2
        CU(cudaStreamWaitEvent(p->stream, p->ev_h2d[s], 0));
        if (i >= 2) CU(cudaStreamWaitEvent(p->stream, p->ev_d2h[s], 0));
        if ((rc = fsp_solve(p, rs[s], ps[s])) != FSP_OK) return rc;
        CU(cudaEventRecord(p->ev_solve[s], p->stream));
        // copy-out of solve i
        CU(cudaStreamWaitEvent(p->s_d2h, p->ev_solve[s], 0));
        CU(cudaMemcpyAsync(phi_hosts[i], ps[s], v * sizeof(double), cudaMemcpyDeviceToHost, p->s_d2h));
        CU(cudaEventRecord(p->ev_d2h[s], p->s_d2h));
    }
    CU(cudaStreamSynchronize(p->s_d2h));
    CU(cudaStreamSynchronize(p->s_h2d));
    CU(cudaStreamSynchronize(p->stream));
    return FSP_OK;
}

int fsp_solve_host_batch(fsp_plan* p, int n, const double* const* rho_hosts, double* const* phi_hosts) {
    if (!p || n < 0 || (n > 0 && (!rho_hosts || !phi_hosts))) return FSP_ERR_INVALID_ARG;
    for (int i = 0; i < n; ++i)
        if (!rho_hosts[i] || !phi_hosts[i]) return FSP_ERR_INVALID_ARG;
    if (!p->precomputed) return FSP_ERR_NOT_PRECOMPUTED;
    if (n == 0) return FSP_OK;
    DeviceGuard dev_guard(p->device);
    const size_t v = user_volume(p);
    int rc;
    if (!p->rho_stage) {
        if ((rc = dev_alloc(&p->rho_stage, v, &p->bytes)) != FSP_OK) return rc;
        if ((rc = dev_alloc(&p->phi_stage, v, &p->bytes)) != FSP_OK) return rc;
    }
    if (!p->rho_stage2) {
        if ((rc = dev_alloc(&p->rho_stage2, v, &p->bytes)) != FSP_OK) return rc;
        if ((rc = dev_alloc(&p->phi_stage2, v, &p->bytes)) != FSP_OK) return rc;
        CU(cudaStreamCreateWithFlags(&p->s_h2d, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&p->s_d2h, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CU(cudaEventCreateWithFlags(&p->ev_h2d[i], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&p->ev_solve[i], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&p->ev_d2h[i], cudaEventDisableTiming));
        }
    }
    rc = batch_pipeline(p, n, rho_hosts, phi_hosts, v);
    if (rc != FSP_OK) {
        // copies to and from the caller's buffers may still be in flight: drain before handing them back
        cudaStreamSynchronize(p->s_h2d); cudaStreamSynchronize(p->stream); cudaStreamSynchronize(p->s_d2h);
        (void)cudaGetLastError();
    }
    return rc;
}

int fsp_solve_field(fsp_plan* p, const double* rho_dev, double* phi_dev, double* E_dev) {
    if (!p || !rho_dev || !E_dev || rho_dev == phi_dev || rho_dev == E_dev) return FSP_ERR_INVALID_ARG;
    if (p->stage != 0) return FSP_ERR_INVALID_ARG;
    if (!p->precomputed) return FSP_ERR_NOT_PRECOMPUTED;
    DeviceGuard dev_guard(p->device);
    const size_t n2 = (size_t)(p->Nx + 1) * 2 * p->Ny * p->Nz, V = user_volume(p);
    int rc;
    if (p->padded) {
        if ((rc = embed_rho(p, rho_dev)) != FSP_OK) return rc;
        rho_dev = p->rho_pad;
    }
    // last pass of one output: straight into the caller's array, or through phi_pad and a crop (R19)
    auto out_x = [&](double* dst, double kder) -> int {
        if (!p->padded) return do_inv_x(p, dst, kder);
        int r = do_inv_x(p, p->phi_pad, kder);
        return r != FSP_OK ? r : crop_out(p, dst);
    };
    if (!p->B3) {   // first field solve of this plan: the buffer that receives the derivative spectra
        double2* b3 = nullptr;
        if ((rc = dev_alloc(&b3, n2, nullptr)) != FSP_OK) return rc;
        if (p->tile_y) {
            const cuuint64_t dims[4] = {(cuuint64_t)2 * p->Nz, 2, (cuuint64_t)p->Ny, (cuuint64_t)(p->Nx + 1)};
            const cuuint64_t strides[3] = {(cuuint64_t)p->Nz * 16, (cuuint64_t)2 * p->Nz * 16, (cuuint64_t)2 * p->Ny * p->Nz * 16};
            const cuuint32_t box[4] = {2 * (cuuint32_t)(p->Ny == 1024 ? 4 : kW), 1, (cuuint32_t)(p->Ny < 256 ? p->Ny : 256), 1};
            if ((rc = make_tensor_map(&p->tmB3y, b3, 4, dims, strides, box)) != FSP_OK) {
                cudaFree(b3);   // B3 stays null: the next call starts over instead of reading through a bad map
                return rc;
            }
        }
        p->B3 = b3;
        p->bytes += n2 * sizeof(double2);
    }
    const int planes = p->Nx + 1;
    const double PI = 3.14159265358979323846;
    // forward passes once: B2 = F_y F_x rho2
    if ((rc = do_fwd_x(p, rho_dev)) != FSP_OK) return rc;
    if ((rc = do_fwd_y(p, 0, p->B2, planes)) != FSP_OK) return rc;
    // The factor -i k_d (R18) commutes with the inverse passes along the other axes, so it is
    // applied in the pass that transforms ITS axis and everything before that pass is shared:
    const double kx = 2.0 * PI / (2.0 * (double)p->Nx * p->h[0]);
    const double ky = 2.0 * PI / (2.0 * (double)p->Ny * p->h[1]);
    const double kz = 2.0 * PI / (2.0 * (double)p->Nz * p->h[2]);
    // E_z: K3 with the factor fused into the spectrum multiply (B2 -> B3), K4, K5
    const DerK kap{0.0, 0.0, kz, p->Nx};
    if ((rc = do_conv_z(p, p->B2, 0, planes, p->B3, &kap)) != FSP_OK) return rc;
    if ((rc = do_inv_y(p, p->B3, p->B1, planes)) != FSP_OK) return rc;
    if ((rc = out_x(E_dev + 2 * V, 0.0)) != FSP_OK) return rc;
    // phi and E_x: plain K3 (in place), K4, then K5 twice on the same B1 (plain, and with -i kx on its input)
    if ((rc = do_conv_z(p, p->B2, 0, planes)) != FSP_OK) return rc;
    if ((rc = do_inv_y(p, p->B2, p->B1, planes)) != FSP_OK) return rc;
    if (phi_dev && (rc = out_x(phi_dev, 0.0)) != FSP_OK) return rc;
    if ((rc = out_x(E_dev, kx)) != FSP_OK) return rc;
    // E_y: K4 with -i ky on its input rows (B2 still holds the output of the plain K3), K5
    if ((rc = do_inv_y(p, p->B2, p->B1, planes, ky)) != FSP_OK) return rc;
    if ((rc = out_x(E_dev + V, 0.0)) != FSP_OK) return rc;
    CU(cudaGetLastError());
    return FSP_OK;
}

int fsp_solve_field_host(fsp_plan* p, const double* rho_host, double* phi_host, double* E_host) {
    if (!p || !rho_host || !E_host) return FSP_ERR_INVALID_ARG;
    if (!p->precomputed) return FSP_ERR_NOT_PRECOMPUTED;
    DeviceGuard dev_guard(p->device);
    const size_t v = user_volume(p);
    int rc;
    if (!p->rho_stage) {
        if ((rc = dev_alloc(&p->rho_stage, v, &p->bytes)) != FSP_OK) return rc;
        if ((rc = dev_alloc(&p->phi_stage, v, &p->bytes)) != FSP_OK) return rc;
    }
    if (!p->E_stage && (rc = dev_alloc(&p->E_stage, 3 * v, &p->bytes)) != FSP_OK) return rc;
    CU(cudaMemcpyAsync(p->rho_stage, rho_host, v * sizeof(double), cudaMemcpyHostToDevice, p->stream));
    if ((rc = fsp_solve_field(p, p->rho_stage, phi_host ? p->phi_stage : nullptr, p->E_stage)) != FSP_OK) return rc;
    if (phi_host) CU(cudaMemcpyAsync(phi_host, p->phi_stage, v * sizeof(double), cudaMemcpyDeviceToHost, p->stream));
    CU(cudaMemcpyAsync(E_host, p->E_stage, 3 * v * sizeof(double), cudaMemcpyDeviceToHost, p->stream));
    CU(cudaStreamSynchronize(p->stream));
    return FSP_OK;
}

double fsp_model_bytes_per_field_solve(const fsp_plan* p, int with_phi) {
    if (!p) return 0.0;
    double k[FSP_NUM_SOLVE_KERNELS];
    fsp_model_bytes_per_solve(p, k);
    return k[0] + k[1] + 2.0 * k[2] + 3.0 * k[3] + (with_phi ? 4.0 : 3.0) * k[4];
}

int fsp_destroy(fsp_plan* p) {
    if (!p) return FSP_ERR_INVALID_ARG;
    DeviceGuard dev_guard(p->device);
    cudaStreamSynchronize(p->stream);
    free_plan_memory(p);
    (void)cudaGetLastError();
    delete p;
    return FSP_OK;
}

size_t fsp_plan_bytes(const fsp_plan* p) { return p ? p->bytes : 0; }
size_t fsp_precompute_peak_bytes(const fsp_plan* p) { return p ? p->peak_transient : 0; }

double fsp_model_bytes_per_solve(const fsp_plan* p, double* per_kernel) {
    if (!p) return 0.0;
    const double V = (double)p->Nx * p->Ny * p->Nz;
    const double H = (double)(p->Nx + 1) * p->Ny * p->Nz;  // complex elements of B1; B2 has 2H
    double k[FSP_NUM_SOLVE_KERNELS];
    k[0] = 8.0 * V + 16.0 * H;                      // K1: read rho, write B1
    k[1] = 16.0 * H + 32.0 * H;                     // K2: read B1, write B2
    // K3: read+write B2, read the unique octant of Ghat (real) once
    k[2] = 32.0 * H + 32.0 * H +
           8.0 * (double)(p->Nx + 1) * (p->Ny + 1) * (p->Nz + 2);
    k[3] = 32.0 * H + 16.0 * H;                     // K4
    k[4] = 16.0 * H + 8.0 * V;                      // K5
    double tot = 0.0;
    for (int i = 0; i < FSP_NUM_SOLVE_KERNELS; ++i) {
        tot += k[i];
        if (per_kernel) per_kernel[i] = k[i];
    }
    return tot;
}

int fsp_get_vg_factors(const fsp_plan* p, int* m_out) {
    if (!p || !m_out) return FSP_ERR_INVALID_ARG;
    if (!p->precomputed) return FSP_ERR_NOT_PRECOMPUTED;
    for (int d = 0; d < 3; ++d) m_out[d] = p->vg_m[d];
    return FSP_OK;
}

int fsp_vg_lattice_is_safe(const fsp_plan* p, int* safe_out) {
    if (!p || !safe_out) return FSP_ERR_INVALID_ARG;
    *safe_out = 1;
    if (p->algorithm == FSP_HOCKNEY || p->algorithm == FSP_VICO_SAFE) return FSP_OK;
    const double Ld[3] = {p->Nx * p->h[0], p->Ny * p->h[1], p->Nz * p->h[2]};
    const double L = p->alpha * std::sqrt(Ld[0] * Ld[0] + Ld[1] * Ld[1] + Ld[2] * Ld[2]);
    for (int d = 0; d < 3; ++d)
        if (4.0 * Ld[d] < L + Ld[d]) *safe_out = 0;
    return FSP_OK;
}

int fsp_get_green_table(const fsp_plan* p, double* T_host) {
    if (!p || !T_host) return FSP_ERR_INVALID_ARG;
    if (!p->precomputed) return FSP_ERR_NOT_PRECOMPUTED;
    DeviceGuard dev_guard(p->device);
    const size_t nt = (size_t)(p->Nx + 1) * (p->Ny + 1) * (p->Nz + 1);
    CU(cudaStreamSynchronize(p->stream));
    if (p->padded) {   // the caller's block (Ux+1)(Uy+1)(Uz+1) of the table of the transform mesh
        std::vector<double> full(nt);
        CU(cudaMemcpy(full.data(), p->T, nt * sizeof(double), cudaMemcpyDeviceToHost));
        for (int i = 0; i <= p->Ux; ++i)
            for (int j = 0; j <= p->Uy; ++j)
                for (int k = 0; k <= p->Uz; ++k)
                    T_host[((size_t)i * (p->Uy + 1) + j) * (p->Uz + 1) + k] = full[((size_t)i * (p->Ny + 1) + j) * (p->Nz + 1) + k];
        return FSP_OK;
    }
    CU(cudaMemcpy(T_host, p->T, nt * sizeof(double), cudaMemcpyDeviceToHost));
    return FSP_OK;
}

int fsp_get_green_spectrum(const fsp_plan* p, double* Ghat_host) {
    if (!p || !Ghat_host) return FSP_ERR_INVALID_ARG;
    if (p->padded) return FSP_ERR_INVALID_ARG;   // the spectrum lives on the transform mesh, not the caller's
    if (!p->precomputed) return FSP_ERR_NOT_PRECOMPUTED;
    DeviceGuard dev_guard(p->device);
    const size_t nt = (size_t)(p->Nx + 1) * (p->Ny + 1) * (p->Nz + 1);
    CU(cudaStreamSynchronize(p->stream));
    CU(cudaMemcpy(Ghat_host, p->Goct, nt * sizeof(double), cudaMemcpyDeviceToHost));
    return FSP_OK;
}

int fsp_set_profiling(fsp_plan* p, int on) {
    if (!p) return FSP_ERR_INVALID_ARG;
    p->profiling = on != 0;
    p->events_used = 0;
    return FSP_OK;
}

int fsp_get_kernel_times(fsp_plan* p, float* ms, int* n_solves) {
    if (!p || !ms || !n_solves) return FSP_ERR_INVALID_ARG;
    DeviceGuard dev_guard(p->device);
    for (int i = 0; i < FSP_NUM_SOLVE_KERNELS; ++i) ms[i] = 0.0f;
    const size_t n = p->events_used / 6;
    if (n > 0) CU(cudaEventSynchronize(p->events[p->events_used - 1]));
    for (size_t s = 0; s < n; ++s)
        for (int i = 0; i < FSP_NUM_SOLVE_KERNELS; ++i) {
            float t = 0.0f;
            CU(cudaEventElapsedTime(&t, p->events[6 * s + i], p->events[6 * s + i + 1]));
            ms[i] += t;
        }
    *n_solves = (int)n;
    p->events_used = 0;
    return FSP_OK;
}


// ---- sharded plan (slab decomposition, shard.cuh) ----------------------------------------------------------
struct fsp_sharded_plan {
    fsp_plan* px = nullptr;    // x stage on the y-slab: mesh (Nx, Ny / P, Nz); its B1 is B1x
    fsp_plan* pyz = nullptr;   // y-z-y middle on this rank's kx planes: mesh (Nx, Ny, Nz); its B1 is B1y
    int rank = 0, nranks = 1, Nx = 0, Ny = 0, Nz = 0, k0 = 0, np = 0;
    double2* peer_b1y[kMaxRanks] = {};   // every rank's B1y (forward transpose target), device-accessible from here
    double2* peer_b1x[kMaxRanks] = {};   // every rank's B1x (backward transpose target)
    bool peers_set = false;
};

static int shard_scatter(fsp_sharded_plan* sp, int direction) {
    ShardCopyArgs a;
    long longest = 0;
    for (int s = 0; s < sp->nranks; ++s) {
        a.dst[s] = direction == 0 ? sp->peer_b1y[s] : sp->peer_b1x[s];
        a.blk[s] = shard_block(sp->Nx, sp->Ny, sp->Nz, sp->nranks, sp->rank, s, direction);
        const long t = a.blk[s].nrun * a.blk[s].run_len;
        if (t > longest) longest = t;
    }
    const double2* src = direction == 0 ? sp->px->B1 : sp->pyz->B1;
    dim3 grid(grid_for(longest, 256), (unsigned)sp->nranks);
    k_shard_copy<<<grid, 256, 0, sp->px->stream>>>(src, a);
    CU(cudaGetLastError());
    return FSP_OK;
}

int fsp_shard_planes(int Nx, int nranks, int rank, int* k0_out, int* np_out) {
    if (Nx < 1 || nranks < 1 || nranks > kMaxRanks || rank < 0 || rank >= nranks || !k0_out || !np_out) return FSP_ERR_INVALID_ARG;
    shard_planes(Nx, nranks, rank, k0_out, np_out);
    return FSP_OK;
}

int fsp_shard_block(int Nx, int Ny, int Nz, int nranks, int src_rank, int dst_rank, int direction, long long* out6) {
    if (Nx < 1 || Ny < 1 || Nz < 1 || nranks < 1 || nranks > kMaxRanks || Ny % nranks != 0 || src_rank < 0 || src_rank >= nranks ||
        dst_rank < 0 || dst_rank >= nranks || (direction != 0 && direction != 1) || !out6)
        return FSP_ERR_INVALID_ARG;
    const ShardBlock b = shard_block(Nx, Ny, Nz, nranks, src_rank, dst_rank, direction);
    out6[0] = b.nrun; out6[1] = b.run_len; out6[2] = b.src_off; out6[3] = b.src_stride; out6[4] = b.dst_off; out6[5] = b.dst_stride;
    return FSP_OK;
}

int fsp_sharded_create(fsp_sharded_plan** out, int Nx, int Ny, int Nz, const double* h, int algorithm, void* cuda_stream,
                       int rank, int nranks) {
    if (!out) return FSP_ERR_INVALID_ARG;
    *out = nullptr;
    auto pow2 = [](int n) { return n >= 8 && (n & (n - 1)) == 0; };
    if (!pow2(Nx) || !pow2(Ny) || !pow2(Nz) || Nx > 1024 || Ny > 1024 || Nz > 1024) return FSP_ERR_INVALID_ARG;
    if (nranks < 1 || nranks > kMaxRanks || rank < 0 || rank >= nranks || Ny % nranks != 0 || Nx + 1 < nranks) return FSP_ERR_INVALID_ARG;
    const long slab_plane = (long)(Ny / nranks) * Nz;   // columns of the x stage
    if (slab_plane < 64) return FSP_ERR_INVALID_ARG;
    fsp_sharded_plan* sp = new (std::nothrow) fsp_sharded_plan();
    if (!sp) return FSP_ERR_OUT_OF_MEMORY;
    sp->rank = rank; sp->nranks = nranks; sp->Nx = Nx; sp->Ny = Ny; sp->Nz = Nz;
    shard_planes(Nx, nranks, rank, &sp->k0, &sp->np);
    // the x stage sees the y-slab as a mesh of its own: K1 and K5 only need Ny_loc * Nz columns of length Nx
    // (K1 and K5 only see "plane = Ny_loc * Nz columns": the slab is handed to them as a mesh Nx x Ny' x Nz' with the
    // same number of columns and both factors powers of two >= 8, whatever Ny / P is)
    const int nz_x = (int)(slab_plane / 8 < 1024 ? slab_plane / 8 : 1024), ny_x = (int)(slab_plane / nz_x);
    int rc = plan_create_impl(&sp->px, Nx, ny_x, nz_x, h, algorithm, cuda_stream, 1, 0, 0);
    if (rc == FSP_OK) rc = plan_create_impl(&sp->pyz, Nx, Ny, Nz, h, algorithm, cuda_stream, 2, sp->k0, sp->np);
    if (rc != FSP_OK) {
        if (sp->px) fsp_destroy(sp->px);
        if (sp->pyz) fsp_destroy(sp->pyz);
        delete sp;
        return rc;
    }
    *out = sp;
    return FSP_OK;
}

int fsp_sharded_set_param(fsp_sharded_plan* sp, int which, double value) {
    if (!sp) return FSP_ERR_INVALID_ARG;
    return fsp_plan_set_param(sp->pyz, which, value);
}

int fsp_sharded_precompute_green(fsp_sharded_plan* sp) {
    if (!sp) return FSP_ERR_INVALID_ARG;
    return fsp_precompute_green(sp->pyz);
}

int fsp_sharded_buffers(const fsp_sharded_plan* sp, void** b1x_out, void** b1y_out, size_t* b1x_bytes, size_t* b1y_bytes) {
    if (!sp || !b1x_out || !b1y_out) return FSP_ERR_INVALID_ARG;
    *b1x_out = sp->px->B1;
    *b1y_out = sp->pyz->B1;
    if (b1x_bytes) *b1x_bytes = sp->px->b1_count * sizeof(double2);
    if (b1y_bytes) *b1y_bytes = sp->pyz->b1_count * sizeof(double2);
    return FSP_OK;
}

int fsp_sharded_set_peers(fsp_sharded_plan* sp, void* const* peer_b1x, void* const* peer_b1y) {
    if (!sp || !peer_b1x || !peer_b1y) return FSP_ERR_INVALID_ARG;
    for (int s = 0; s < sp->nranks; ++s) {
        if (!peer_b1x[s] || !peer_b1y[s]) return FSP_ERR_INVALID_ARG;
        sp->peer_b1x[s] = static_cast<double2*>(peer_b1x[s]);
        sp->peer_b1y[s] = static_cast<double2*>(peer_b1y[s]);
    }
    if (sp->peer_b1x[sp->rank] != sp->px->B1 || sp->peer_b1y[sp->rank] != sp->pyz->B1) return FSP_ERR_INVALID_ARG;
    sp->peers_set = true;
    return FSP_OK;
}

int fsp_sharded_solve_phase(fsp_sharded_plan* sp, int phase, const double* rho_slab_dev, double* phi_slab_dev) {
    if (!sp || phase < 0 || phase > 2) return FSP_ERR_INVALID_ARG;
    if (!sp->peers_set) return FSP_ERR_INVALID_ARG;
    if (!sp->pyz->precomputed) return FSP_ERR_NOT_PRECOMPUTED;
    DeviceGuard dev_guard(sp->px->device);
    int rc;
    if (phase == 0) {          // K1 on the y-slab, then the forward transpose into every rank's B1y
        if (!rho_slab_dev) return FSP_ERR_INVALID_ARG;
        if ((rc = do_fwd_x(sp->px, rho_slab_dev)) != FSP_OK) return rc;
        return shard_scatter(sp, 0);
    }
    if (phase == 1) {          // K2, K3, K4 on this rank's kx planes, then the backward transpose into every rank's B1x
        fsp_plan* q = sp->pyz;
        if ((rc = do_fwd_y(q, 0, q->B2, sp->np)) != FSP_OK) return rc;
        if ((rc = do_conv_z(q, q->B2, 0, sp->np)) != FSP_OK) return rc;
        if ((rc = do_inv_y(q, q->B2, q->B1, sp->np)) != FSP_OK) return rc;
        return shard_scatter(sp, 1);
    }
    if (!phi_slab_dev) return FSP_ERR_INVALID_ARG;
    if ((rc = do_inv_x(sp->px, phi_slab_dev)) != FSP_OK) return rc;   // K5 on the y-slab
    CU(cudaGetLastError());
    return FSP_OK;
}

size_t fsp_sharded_bytes(const fsp_sharded_plan* sp) { return sp ? sp->px->bytes + sp->pyz->bytes : 0; }

int fsp_sharded_destroy(fsp_sharded_plan* sp) {
    if (!sp) return FSP_ERR_INVALID_ARG;
    fsp_destroy(sp->px);
    fsp_destroy(sp->pyz);
    delete sp;
    return FSP_OK;
}

// thin wrappers over the CUDA IPC calls, so that one-process-per-GPU launches can exchange the workspace addresses that
// fsp_sharded_set_peers needs (handle: 64 bytes, sent between ranks by the caller, e.g. torch.distributed all_gather)
int fsp_ipc_get_handle(void* dev_ptr, void* handle64_out) {
    if (!dev_ptr || !handle64_out) return FSP_ERR_INVALID_ARG;
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "handle size");
    CU(cudaIpcGetMemHandle(static_cast<cudaIpcMemHandle_t*>(handle64_out), dev_ptr));
    return FSP_OK;
}
int fsp_ipc_open_handle(const void* handle64, void** dev_ptr_out) {
    if (!handle64 || !dev_ptr_out) return FSP_ERR_INVALID_ARG;
    cudaIpcMemHandle_t hnd;
    std::memcpy(&hnd, handle64, sizeof(hnd));
    CU(cudaIpcOpenMemHandle(dev_ptr_out, hnd, cudaIpcMemLazyEnablePeerAccess));
    return FSP_OK;
}
int fsp_ipc_close_handle(void* dev_ptr) {
    if (!dev_ptr) return FSP_ERR_INVALID_ARG;
    CU(cudaIpcCloseMemHandle(dev_ptr));
    return FSP_OK;
}

}  // extern "C"

// ---- fp64 issue-cost micro-benchmark (include/fsp.h: fsp_ubench_fp64; ubench.cuh) ------------------------------------
extern "C" int fsp_ubench_fp64(int mode, int warps_per_sm, double* clk_per_instr_out) {
    if (!clk_per_instr_out || mode < 0 || mode > 3) return FSP_ERR_INVALID_ARG;
    if (warps_per_sm < 4 || warps_per_sm > 32 || warps_per_sm % 4 != 0) return FSP_ERR_INVALID_ARG;
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int threads = warps_per_sm * 32, iters = 4096;
    double *out = nullptr, *in = nullptr;
    long long* clk = nullptr;
    int rc = dev_alloc(&out, (size_t)sms * threads, nullptr);
    if (rc == FSP_OK) rc = dev_alloc(&in, (size_t)threads + 48, nullptr);
    if (rc == FSP_OK) rc = dev_alloc(&clk, 1, nullptr);
    long long h = 0;
    if (rc == FSP_OK) {
        cudaMemset(in, 0, sizeof(double) * ((size_t)threads + 48));
        for (int rep = 0; rep < 2; ++rep) {   // the second launch is the measurement (the first loads the code)
            switch (mode) {
                case 0: k_ubench_fp64<0><<<sms, threads>>>(out, in, iters, clk); break;
                case 1: k_ubench_fp64<1><<<sms, threads>>>(out, in, iters, clk); break;
                case 2: k_ubench_fp64<2><<<sms, threads>>>(out, in, iters, clk); break;
                default: k_ubench_fp64<3><<<sms, threads>>>(out, in, iters, clk); break;
            }
        }
        cudaError_t e = cudaDeviceSynchronize();
        if (e == cudaSuccess) e = cudaMemcpy(&h, clk, sizeof(h), cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) { (void)cudaGetLastError(); rc = map_cuda(e); }
    }
    cudaFree(out); cudaFree(in); cudaFree(clk);
    if (rc != FSP_OK) return rc;
    // per scheduler (4 per SM): warps_per_sm / 4 warps each issue iters * 16 instructions
    *clk_per_instr_out = (double)h / ((double)iters * 16.0 * (warps_per_sm / 4.0));
    return FSP_OK;
}

// ---- the allocation-free entry point (include/fsp.h: fsp_green_spectrum_static) -------------------------------------
// The scratch of the 3-D DCT-I (the array between the y pass and the x pass) as a file-scope device array.  In HOST code
// the name g_static_scratch is a stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) double g_static_scratch[FSP_STATIC_MAX_DOUBLES];

namespace {
constexpr int kStaticMaxDevices = 64;
std::atomic<double*> g_static_scratch_ptr[kStaticMaxDevices];   // zero-initialised: not yet resolved on that device

int static_scratch_address(double** out) {
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return FSP_ERR_NO_DEVICE;
    double* ptr = g_static_scratch_ptr[dev].load(std::memory_order_acquire);
    if (!ptr) {   // (two threads may both resolve it: same answer, no allocation either way)
        CU(cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_static_scratch));
        if (!ptr) return FSP_ERR_CUDA;
        g_static_scratch_ptr[dev].store(ptr, std::memory_order_release);
    }
    *out = ptr;
    return FSP_OK;
}

// one pass of cosine sums over an nA x nB grid of pencils (strides as in dct1_strided); n <= 512: 25 KB of shared memory
// at most, below the 48 KB that need no opt-in.
// C = 4 on purpose: the instantiation must be one that the plan path (dct1_strided: C = 8) never launches.  That path
// sets cudaFuncAttributeMaxDynamicSharedMemorySize of ITS kernel to the largest request seen so far, which LOWERS the
// limit below the default 48 KB while only short transforms have run -- a launch from here with a longer one would then
// fail, or not, depending on which plans the process has created before.  This kernel's attribute is never touched.
int static_dct1_pass(const double* in, double* out, int n, long nA, long nB, const long ai[3], const long ao[3],
                     cudaStream_t stream) {
    constexpr int C = 4;
    const size_t smem = sizeof(double) * ((size_t)2 * n + (size_t)(n + 1) * C);
    k_dct1_direct<C, false><<<(unsigned)(nA * ((nB + C - 1) / C)), 256, smem, stream>>>(
        in, out, n, n + 1, nB, ai[0], ai[1], ai[2], ao[0], ao[1], ao[2], 1.0, GLFill{0.0, 0.0, 0.0, 0.0, 0});
    CU(cudaGetLastError());
    return FSP_OK;
}
}  // namespace

extern "C" int fsp_green_spectrum_static(const double* T_dev, double* Ghat_dev, int Nx, int Ny, int Nz, void* cuda_stream) {
    if (!T_dev || !Ghat_dev || T_dev == Ghat_dev) return FSP_ERR_INVALID_ARG;
    if (Nx < 1 || Ny < 1 || Nz < 1 || Nx > 512 || Ny > 512 || Nz > 512) return FSP_ERR_INVALID_ARG;
    const long X = Nx + 1L, Y = Ny + 1L, Z = Nz + 1L;
    if (X * Y * Z > (long)FSP_STATIC_MAX_DOUBLES) return FSP_ERR_STATIC_CAPACITY;
    double* mid = nullptr;
    int rc = static_scratch_address(&mid);
    if (rc != FSP_OK) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    {   // z pass: T[x][y][z] -> Ghat[x][y][kz]
        const long ai[3] = {Y * Z, Z, 1}, ao[3] = {Y * Z, Z, 1};
        if ((rc = static_dct1_pass(T_dev, Ghat_dev, Nz, X, Y, ai, ao, stream)) != FSP_OK) return rc;
    }
    {   // y pass: Ghat[x][y][kz] -> mid[ky][x][kz]  (ky outermost: the x pass reads pencils Z doubles apart)
        const long ai[3] = {Y * Z, 1, Z}, ao[3] = {Z, 1, X * Z};
        if ((rc = static_dct1_pass(Ghat_dev, mid, Ny, X, Z, ai, ao, stream)) != FSP_OK) return rc;
    }
    {   // x pass: mid[ky][x][kz] -> Ghat[kx][ky][kz]
        const long ai[3] = {X * Z, 1, Z}, ao[3] = {Z, 1, Y * Z};
        if ((rc = static_dct1_pass(mid, Ghat_dev, Nx, Y, Z, ai, ao, stream)) != FSP_OK) return rc;
    }
    return FSP_OK;
}

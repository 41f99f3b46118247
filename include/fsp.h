/*
 * fsp.h -- C ABI of the B200-native free-space Poisson convolution library (libfsp.so).
 *
 * The hot path of arxiv 2405.02603 (cited as PAPER.md:<line>):
 *
 *     phi = hx hy hz * F^-1{ F{rho2} x F{G2} } restricted to the physical mesh
 *
 * with rho2 the zero-padded source on the doubled grid and G2 the mirrored,
 * periodic Green's function of either
 *     FSP_HOCKNEY : G = 1/(4 pi |x|), origin regularised
 *     FSP_VICO    : truncated-kernel spectrum Eq. 3, inverse FFT on the 4N grid, restricted
 *
 *     FSP_VICO_2  : same values from the (2N+1)^3 grid with a DCT-I
 *     FSP_VICO_SAFE : FSP_VICO_2 with per-axis oversampling, safe on elongated boxes (see the enum)
 * (names as PAPER.md:199: HOCKNEY / VICO / VICO_2).
 *
 * Everything behind these calls runs in hand-written sm_100a CUDA kernels: no FFT library, no CPU
 * fallback.  One GPU, one plan = one mesh; fp64 throughout.  eps0 = 1: the caller divides by eps0.
 *
 * Conventions
 *   - Mesh Nx x Ny x Nz, spacings h[0..2] = hx, hy, hz, 2 <= N_d <= 1024.  Transform lengths
 *     are 2^k (the paper's sizes all are), 3 2^k and 5 2^k between 8 and 1024 (Nz a multiple
 *     of 8): on such a mesh nothing is embedded and every algorithm gives the paper's result for the caller's
 *     mesh.  A mesh with another N_d is embedded in the next such mesh N'_d >= max(N_d, 8) (zero density
 *     outside, result cropped; R19).  The cyclic convolution is exact for any period >= 2 N_d - 1,
 *     so FSP_HOCKNEY still gives the paper's result for the caller's mesh; the Vico-Greengard table is then
 *     that of the enclosing box N'_d h_d (a larger truncation radius L, same free-space kernel); the spectral
 *     gradient of fsp_solve_field has period 2 N'_d h_d.  Cost and memory are those of the N' mesh.
 *     (FSP_VICO, the plain 4x-oversampled precompute, takes power-of-two transform meshes only: every other
 *     mesh is embedded in the next power of two.)
 *   - rho, phi: dense fp64 arrays of shape (Nx, Ny, Nz) in C order, index (ix*Ny + iy)*Nz + iz,
 *     iz fastest.  The sample position inside a cell does not matter (translation invariance).
 *   - "dev" pointers are CUDA device pointers on the device that was current at plan creation (the
 *     plan's device); "host" pointers are ordinary host memory (pinned memory makes the copies
 *     asynchronous).  Devices: every call that touches the GPU switches to the plan's device for its
 *     duration and restores the caller's current device before it returns, so plans on several devices can
 *     be driven from one process and one thread whatever device is current; shared-memory opt-ins and
 *     occupancies are cached per device.  Threads: different plans may be used from different host
 *     threads concurrently; one plan must not be used by two threads at the same time.
 *   - The caller owns rho and phi; rho is read-only; rho and phi must not overlap.  The plan owns
 *     the spectrum, twiddle tables and workspace.  fsp_solve allocates nothing and does not
 *     synchronise the host: it is ordered on the stream given at plan creation.
 *   - Every call returns FSP_OK (0) or a negative error code; nothing throws or aborts across
 *     the ABI.  A plan pointer that is NULL gives FSP_ERR_INVALID_ARG.
 */
#ifndef FSP_H
#define FSP_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fsp_plan fsp_plan; /* opaque, library-owned */

/* algorithm */
enum {
    FSP_HOCKNEY = 0,
    FSP_VICO = 1,
    FSP_VICO_2 = 2,
    /* FSP_VICO_2 with per-axis oversampling factors m_d instead of the paper's 4: m_d = 4,
     * doubled while m_d < 1 + L / L_d, L = alpha * box diagonal, L_d = N_d h_d.  The kernel
     * truncated at radius L is periodised with period m_d L_d and used up to displacement L_d, so its
     * images stay out of the table iff m_d L_d >= L + L_d; with m = 4 that fails on boxes longer than
     * about 2.7 times their shortest side (the paper's beam-dynamics use case).  Identical to
     * FSP_VICO_2 whenever the rule gives (4,4,4), e.g. on every cube.  DESIGN.md reading R17. */
    FSP_VICO_SAFE = 3
};

/* error codes */
enum {
    FSP_OK = 0,
    FSP_ERR_INVALID_ARG = -1,     /* null pointer, N_d outside [2,1024], h <= 0, bad enum             */
    FSP_ERR_NOT_PRECOMPUTED = -2, /* fsp_solve / getters before fsp_precompute_green                 */
    FSP_ERR_OUT_OF_MEMORY = -3,   /* device allocation failed (e.g. FSP_VICO at 1024^3: (4N)^3 lattice) */
    FSP_ERR_CUDA = -4,            /* a CUDA runtime call or kernel launch failed                     */
    FSP_ERR_NO_DEVICE = -5,       /* no CUDA device / not an sm_100 device                           */
    FSP_ERR_STATIC_CAPACITY = -6  /* fsp_green_spectrum_static: table larger than FSP_STATIC_MAX_DOUBLES */
};

/* parameters settable before fsp_precompute_green */
enum {
    FSP_PARAM_G0 = 0,    /* HE value at the origin, default +1/(4 pi)  (R5) */
    FSP_PARAM_ALPHA = 1, /* VG window factor, default 1.1; must be > 1 (L = alpha x diagonal
                            has to exceed the largest displacement), else FSP_ERR_INVALID_ARG       */
    FSP_PARAM_CHUNK_PLANES = 2, /* kx-planes per pass of the y-z-y middle (0 = all at once); takes
                                  effect at the next fsp_solve; does not change results             */
    FSP_PARAM_K2_VARIANT = 4, /* kernel of the forward y pass at Ny = 512 (kept for A/B measurements): 0 (default) = the
                                zero-padded column of 2 Ny points in one group (k_fwd_y_f); 1 = two half-length
                                branches in two groups (k_fwd_y_t).  Takes effect at the next fsp_solve          */
    FSP_PARAM_PERIODIC = 5, /* periodic directions (PAPER.md:67 step 1: only "the non-periodic directions (those which have
                              open boundary conditions)" are doubled; reading R20).  value = bit
                              mask, 1: x, 2: y, 4: z; default 0 = all open (the paper's configurations).  Along a periodic
                              direction d the result is the CYCLIC convolution of period N_d with the kernel made periodic
                              by "circular shifting": G at the nearest image, displacement
                              min(|i - j|, N_d - |i - j|) h_d; rho is taken as N_d-periodic there, nothing is padded.
                              (The nearest image only: the lattice sum of 1/r over all images does not converge and the
                              paper gives no other rule.)  FSP_HOCKNEY only, and only on meshes that are transformed at
                              their own size (2^k, 3 2^k, 5 2^k), else FSP_ERR_INVALID_ARG.  Same five kernels and the same
                              cost as the open solve: the periodic kernel's spectrum on the doubled grid has zero odd bins
                              (a periodic z with Nz = 2^k is cheaper, see FSP_PARAM_PERIODIC_FAST_Z).
                              fsp_get_green_table then returns the folded table T'[i] = T[min(i, N_d - i)].  Invalidates
                              the spectrum: call fsp_precompute_green again                                        */
    FSP_PARAM_PERIODIC_FAST_Z = 6, /* 1 (default): a periodic z direction with Nz a power of two runs the z pass on Nz-point
                                     transforms (k_conv_z_periodic: the saving PAPER.md:67's step 1 implies, along z);
                                     0: the doubled-grid kernel as for every other case.  Same result to rounding; takes
                                     effect at the next fsp_solve (fsp_solve_field always uses the doubled-grid kernels) */
    FSP_PARAM_K3_VARIANT = 3  /* kernel of the z pass (kept for A/B measurements).  0 (default): the whole zero-padded
                                pencil in one lane group (k_conv_z_f, Nz = 256, 512; the prime-factor kernel
                                k_conv_z_pf at Nz = 96, 192, 384; k_conv_z_g2 at the other 3 * 2^k, 5 * 2^k).  1: two
                                half-length branches (k_conv_z_p, k_conv_z_g).  2: Nz = 512: the pair scheme with 32
                                lanes per branch (k_conv_z_s); Nz = 96, 192, 384: k_conv_z_g2.  Invalidates the
                                spectrum (its row layout follows the kernel): call fsp_precompute_green again.
                                Results agree to rounding, all within the tolerances of DESIGN.md       */
};

/* number of kernels one fsp_solve launches (the five passes of DESIGN.md "The path") */
#define FSP_NUM_SOLVE_KERNELS 5

/*
 * plan(Nx,Ny,Nz,h,algorithm)  -- PAPER.md:65 (mesh and spacings), :199 (algorithm).
 *   out          host pointer receiving the new plan
 *   h            host pointer to 3 doubles, all > 0
 *   cuda_stream  a cudaStream_t (0/NULL = the legacy default stream); all work of this plan is
 *                enqueued there
 * Allocates the workspace of the solve (two complex intermediates) and the spectrum.  Does not
 * touch the Green's function: call fsp_precompute_green next.
 */
int fsp_plan_create(fsp_plan** out, int Nx, int Ny, int Nz, const double* h, int algorithm,
                    void* cuda_stream);

/* Set FSP_PARAM_* (only effective before the next fsp_precompute_green). */
int fsp_plan_set_param(fsp_plan* p, int which, double value);

/*
 * New mesh spacings for an existing plan (same Nx, Ny, Nz) -- PAPER.md:98: the Green's function is
 * reused "as long as the mesh spacing does not change"; when the domain follows the bunch it does
 * change, and only the precompute has to be redone: workspace, tables and tensor maps are kept.
 * Invalidates the spectrum: fsp_solve returns FSP_ERR_NOT_PRECOMPUTED until fsp_precompute_green
 * has been called again.  h: host pointer to 3 doubles, all > 0.
 */
int fsp_plan_set_spacing(fsp_plan* p, const double* h);

/*
 * precompute_green(plan) -- PAPER.md:72-76 (HE), :88-98 (VG), :100-102 (VG modified); "calculated
 * ... in only one pre-computation step ... reused every time step".
 * Fills the plan-owned real-space table T[dx][dy][dz] (0 <= d_d <= N_d, the kernel at displacement
 * (dx hx, dy hy, dz hz)) and the spectrum F{G2} of its 8-case mirror, with the
 * factor hx hy hz / (8 Nx Ny Nz) of PAPER.md:80 folded in.  Transient device memory is allocated
 * and freed inside the call (FSP_VICO: the C2R half spectrum of the (4N)^3 lattice, (2Nx+1)(4Ny)(4Nz) complex
 * values, 8.6 GB at 256^3; FSP_VICO_2: (2Nx+1)(2Ny+1)(2Nz+1) reals).  Synchronises the
 * stream before returning.  Re-callable (e.g. after fsp_plan_set_param).
 */
int fsp_precompute_green(fsp_plan* p);

/*
 * solve(plan, rho, phi) -- PAPER.md:67-82 steps 1-5 as five fused/pruned kernel launches.
 *   rho_dev  device pointer, Nx*Ny*Nz doubles, read-only
 *   phi_dev  device pointer, Nx*Ny*Nz doubles, overwritten
 * Asynchronous with respect to the host.
 */
int fsp_solve(fsp_plan* p, const double* rho_dev, double* phi_dev);

/*
 * The same solve from HOST buffers: copies rho host->device, runs the five kernels, copies phi
 * device->host, then synchronises the stream.  Uses plan-owned staging buffers (allocated on first
 * use).  With pinned host memory the copies are true asynchronous DMA transfers.
 */
int fsp_solve_host(fsp_plan* p, const double* rho_host, double* phi_host);

/*
 * n solves from HOST buffers as a pipeline: while solve i runs, rho of solve i+1 is copied in and phi of
 * solve i-1 is copied out, on two copy streams of the plan and two pairs of plan-owned staging buffers
 * (PCIe is full duplex, and the copies take about three times as long as the five kernels).  Every
 * solve still has its input copied host->device and its result copied device->host inside the call; the
 * results are identical to n calls of fsp_solve_host.  For independent densities (bunches, time slices
 * already on the host); pointers may repeat.  Needs pinned host memory to overlap.  Synchronises all
 * three streams before returning.
 *   rho_hosts, phi_hosts  host arrays of n host pointers, each to Nx*Ny*Nz doubles
 */
int fsp_solve_host_batch(fsp_plan* p, int n, const double* const* rho_hosts, double* const* phi_hosts);

/*
 * Field output -- PAPER.md:227-231, Eq. A.1: "the electric field E(x) is obtained from E = -grad phi".
 * The paper does not say how the gradient is taken; here it is taken where the solver already is, in
 * Fourier space on the doubled grid (reading R18):
 *     E_d = -hx hy hz F^-1{ i k_d F{rho2} x F{G2} } restricted,  k_d = 2 pi m'_d / (2 N_d h_d),
 * m' the signed mode number, zero at the Nyquist index m = N_d.  This keeps the accuracy class of the
 * Green's function: second order for FSP_HOCKNEY, spectral for the Vico-Greengard algorithms.
 *   rho_dev  device pointer, Nx*Ny*Nz doubles, read-only
 *   phi_dev  device pointer, Nx*Ny*Nz doubles, or NULL if the potential is not wanted
 *   E_dev    device pointer, 3*Nx*Ny*Nz doubles, component-major: E_dev[d*V + (ix*Ny+iy)*Nz+iz], d = x,y,z
 * The factor -i k_d is fused into the pass that transforms axis d (the spectrum multiply of the middle
 * pass for z, the input of the inverse y pass, the input of the inverse x pass), and everything before
 * that pass is shared: 2 forward + 2 middle + 3 inverse-y + 3 (+1 for phi) inverse-x launches.  The first
 * call allocates one more plan-owned intermediate the size of the larger workspace array (counted by
 * fsp_plan_bytes from then on).  FSP_PARAM_CHUNK_PLANES does not apply.  Asynchronous like fsp_solve.
 */
int fsp_solve_field(fsp_plan* p, const double* rho_dev, double* phi_dev, double* E_dev);

/* The same from HOST buffers (phi_host may be NULL); synchronises the stream before returning. */
int fsp_solve_field_host(fsp_plan* p, const double* rho_host, double* phi_host, double* E_host);

/* Frees everything the plan owns (synchronises its stream first). */
int fsp_destroy(fsp_plan* p);

/* ---- slab decomposition over several GPUs -----------------------------------------------------
 * the paper runs its large meshes on many GPUs (heFFTe pencils, MPI all-to-all).  Here one solve
 * is split over P GPUs with ONE global transpose each way:
 *   rank r owns the y-slab rho_r[x][yl][z], yl < Ny/P, and the same slab of phi;
 *   phase 0: K1 (R2C along x) on the slab, then every rank writes, through peer memory (NVLink P2P stores, no pack
 *            buffer), the kx planes [k0_s, k0_s + np_s) of its result into rank s's y-z workspace B1y_s[kxl][y][z];
 *   phase 1: K2, K3, K4 on the rank's own kx planes (spectrum rows of those planes only), then the transpose back
 *            into every rank's x workspace B1x_r[kx][yl][z];
 *   phase 2: K5 (C2R along x) on the slab.
 * Between phases ALL ranks must have finished the previous phase (the caller synchronises its stream and runs a
 * barrier, e.g. torch.distributed.barrier(); two barriers per solve, nothing else crosses ranks).  Bytes leaving a GPU
 * per solve: 2 x 16 (Nx+1)(Ny/P) Nz (P-1)/P.  Power-of-two meshes with Ny % P == 0, P <= 16, (Ny/P) Nz >= 64.
 * The Green precompute is replicated: every rank computes the whole table and octant (2 x 8 (N+1)^3 bytes, allocated
 * for the duration of fsp_sharded_precompute_green only and reported by its peak) and keeps the spectrum rows of its
 * own planes; between solves a rank holds its slab of the workspace and those rows, nothing of full size.
 * Verified on ONE device with P plans in one process (phases run in turn, tests/test_gpu_sharded.py) and, for the
 * index arithmetic, by a world-size-2 CPU test; NOT yet measured on a multi-GPU node.
 */
typedef struct fsp_sharded_plan fsp_sharded_plan;

/* kx planes [*k0_out, *k0_out + *np_out) of rank `rank`: contiguous slabs of the Nx + 1 planes. */
int fsp_shard_planes(int Nx, int nranks, int rank, int* k0_out, int* np_out);

/* The block rank src_rank sends to dst_rank (direction 0: forward transpose B1x -> B1y; 1: backward B1y -> B1x) as
 * out6 = {nrun, run_len, src_off, src_stride, dst_off, dst_stride} in complex (16-byte) elements: run i covers
 * src[src_off + i src_stride + j] -> dst[dst_off + i dst_stride + j], j < run_len.  Host only (no GPU needed). */
int fsp_shard_block(int Nx, int Ny, int Nz, int nranks, int src_rank, int dst_rank, int direction, long long* out6);

/* plan for rank `rank` of `nranks` on the current device; stream as in fsp_plan_create. */
int fsp_sharded_create(fsp_sharded_plan** out, int Nx, int Ny, int Nz, const double* h, int algorithm,
                       void* cuda_stream, int rank, int nranks);
int fsp_sharded_set_param(fsp_sharded_plan* sp, int which, double value);
int fsp_sharded_precompute_green(fsp_sharded_plan* sp);

/* Device pointers (and sizes) of this rank's two transpose targets; the caller makes them known to every rank
 * (same process: the pointers themselves; one process per GPU: fsp_ipc_get_handle / fsp_ipc_open_handle). */
int fsp_sharded_buffers(const fsp_sharded_plan* sp, void** b1x_out, void** b1y_out, size_t* b1x_bytes, size_t* b1y_bytes);

/* peer_b1x[s], peer_b1y[s]: addresses, valid on THIS device, of rank s's buffers, s < nranks (own entries included). */
int fsp_sharded_set_peers(fsp_sharded_plan* sp, void* const* peer_b1x, void* const* peer_b1y);

/* One phase (0, 1, 2; see above) of one solve, asynchronous on the plan's stream.  rho_slab_dev (phase 0) and
 * phi_slab_dev (phase 2): Nx * (Ny/P) * Nz doubles, [x][yl][z]; ignored in the other phases. */
int fsp_sharded_solve_phase(fsp_sharded_plan* sp, int phase, const double* rho_slab_dev, double* phi_slab_dev);

size_t fsp_sharded_bytes(const fsp_sharded_plan* sp);
int fsp_sharded_destroy(fsp_sharded_plan* sp);

/* cudaIpcGetMemHandle / cudaIpcOpenMemHandle / cudaIpcCloseMemHandle on 64-byte handles (host pointers). */
int fsp_ipc_get_handle(void* dev_ptr, void* handle64_out);
int fsp_ipc_open_handle(const void* handle64, void** dev_ptr_out);
int fsp_ipc_close_handle(void* dev_ptr);

/* ---- queries and test hooks (no hot-path cost) ------------------------------------------------ */

/* Device bytes the plan holds between solves (workspace + spectrum + tables [+ staging]). */
size_t fsp_plan_bytes(const fsp_plan* p);

/* Largest transient device allocation made by the last fsp_precompute_green. */
size_t fsp_precompute_peak_bytes(const fsp_plan* p);

/* Algorithmic (minimal-traffic) HBM bytes of one solve: total, and per kernel
 * if per_kernel (host pointer to FSP_NUM_SOLVE_KERNELS doubles) is not NULL. */
double fsp_model_bytes_per_solve(const fsp_plan* p, double* per_kernel);

/* Algorithmic HBM bytes of one fsp_solve_field: K1 + K2 + 2 K3 + 3 K4 + (3 or 4) K5 in the per-kernel
 * figures of fsp_model_bytes_per_solve (4 K5 if with_phi != 0). */
double fsp_model_bytes_per_field_solve(const fsp_plan* p, int with_phi);

/* Oversampling factors (m_x, m_y, m_z) used by the last fsp_precompute_green of a VG algorithm
 * (4,4,4 for FSP_VICO and FSP_VICO_2); m_out: host pointer to 3 ints. */
int fsp_get_vg_factors(const fsp_plan* p, int* m_out);

/* Does the frequency lattice of the plan's Vico-Greengard algorithm keep the periodic images of the truncated kernel
 * out of the table?  PAPER.md:92-94: L = alpha x diagonal and a fixed 4x oversampling; the kernel of radius L is
 * periodised with period m_d L_d and used up to displacement L_d, so the condition is m_d L_d >= L + L_d on every
 * axis (R17).  *safe_out = 1 if it holds for the factors the plan would use NOW (m = 4 for FSP_VICO and
 * FSP_VICO_2; the per-axis factors of FSP_VICO_SAFE, which satisfy it by construction; FSP_HOCKNEY: always 1), else
 * 0: on such a box (longer than about 2.7 times its shortest side) FSP_VICO / FSP_VICO_2 alias silently and
 * FSP_VICO_SAFE is the algorithm to use.  No GPU work; callable before fsp_precompute_green. */
int fsp_vg_lattice_is_safe(const fsp_plan* p, int* safe_out);

/* Copies the real-space table T, (Nx+1)(Ny+1)(Nz+1) doubles in C order, to host memory. */
int fsp_get_green_table(const fsp_plan* p, double* T_host);

/* Copies the unique octant of the un-normalised spectrum F{G2}[kx][ky][kz], 0 <= k_d <= N_d,
 * (Nx+1)(Ny+1)(Nz+1) doubles in C order (F{G2} is real and even), to host memory.  Power-of-two meshes
 * only: on an embedded mesh the spectrum belongs to the transform mesh (FSP_ERR_INVALID_ARG). */
int fsp_get_green_spectrum(const fsp_plan* p, double* Ghat_host);

/*
 * spectrum_static(T) -- the last step of the Green precompute, T -> F{G2} octant, WITHOUT any allocation.
 *
 * For callers that cannot call cudaMalloc where the spectrum has to be refreshed (the spacing changes whenever the bunch
 * moves): under CUDA graph capture, in a serving loop, in harnesses that forbid it.  Computes what
 * fsp_precompute_green leaves behind fsp_get_green_spectrum,
 *     Ghat[kx][ky][kz] = sum_d w_dx w_dy w_dz T[dx][dy][dz] cos(pi kx dx/Nx) cos(pi ky dy/Ny) cos(pi kz dz/Nz),
 * w = 1 at d = 0 and d = N_d, 2 between -- the 3-D DCT-I of the table, which IS the DFT of the mirrored G2
 * (G2 is real and even) -- as three passes of cosine sums (k_dct1_direct, any N_d).
 *   T_dev      device pointer, (Nx+1)(Ny+1)(Nz+1) doubles in C order (the layout of fsp_get_green_table); read-only
 *   Ghat_dev   device pointer, same shape; written; must not overlap T_dev.  Both on the CURRENT device
 *   Nx,Ny,Nz   1 <= N_d <= 512 and (Nx+1)(Ny+1)(Nz+1) <= FSP_STATIC_MAX_DOUBLES (a 64^3 mesh: 65^3 entries);
 *              a larger table gives FSP_ERR_STATIC_CAPACITY and launches nothing
 *   cuda_stream  the three kernels are enqueued there; no host synchronisation
 * Scratch: the intermediate between the second and the third pass lives in a file-scope `static __device__` array of
 * FSP_STATIC_MAX_DOUBLES doubles (2.2 MB) that every GPU holds from the moment it loads libfsp.so until the process
 * exits.  No cudaMalloc, cudaFree or allocating library call is made, on the first call or later (the first call on a
 * device resolves the array's device address with cudaGetSymbolAddress: make one call before starting a capture).
 * ALL calls on one device share that array: two calls that overlap on the GPU (different streams, or graphs replayed
 * concurrently) race and give garbage; calls on one stream are ordered and safe.  The array keeps the last call's
 * contents; nothing in it has to start at zero (every entry that is read was written by the same call's second pass).
 */
#define FSP_STATIC_MAX_DOUBLES 274625 /* 65^3 */
int fsp_green_spectrum_static(const double* T_dev, double* Ghat_dev, int Nx, int Ny, int Nz, void* cuda_stream);

/*
 * Per-kernel timing.  With profiling on, fsp_solve brackets each of its kernels with CUDA events
 * on the plan's stream; fsp_get_kernel_times synchronises those events and returns, per kernel,
 * the SUM of durations in milliseconds over all solves since the last reset (ms, host pointer to
 * FSP_NUM_SOLVE_KERNELS floats) and the number of solves summed (n_solves).  Resets the sums.
 */
int fsp_set_profiling(fsp_plan* p, int on);
int fsp_get_kernel_times(fsp_plan* p, float* ms, int* n_solves);

/*
 * Measurement hook (bench.py): clocks per fp64 warp-instruction and scheduler on the current
 * device, with warps_per_sm (4, 8, .. 32) resident warps per SM each issuing a stream of independent instructions.
 *   mode 0  DFMA, three register sources, none shared with the instruction before   (B200: 3.0)
 *   mode 1  DFMA, two sources repeated from the instruction before (operand reuse)    (2.2)
 *   mode 2  DFMA, one source repeated                                                 (2.2)
 *   mode 3  DADD, two register sources                                                (2.0)
 * clk_per_instr_out: host pointer.  Allocates and frees three small device buffers; synchronises the device.
 */
int fsp_ubench_fp64(int mode, int warps_per_sm, double* clk_per_instr_out);

/* Name of solve kernel i (0..FSP_NUM_SOLVE_KERNELS-1), static string. */
const char* fsp_kernel_name(int i);

/* Static description of an error code. */
const char* fsp_strerror(int code);

/* Library version (major*100 + minor). */
int fsp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* FSP_H */

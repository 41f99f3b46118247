// shard.cuh -- slab decomposition of one solve over P GPUs (the paper runs its
// 512^3 .. 1024^3 meshes on many GPUs with heFFTe pencils and MPI all-to-all).  Here: ONE global transpose each way.
//
//   rank r owns the y-slab  rho_r[x][yl][z],  yl < Ny/P  (y = r Ny/P + yl)           -> K1 along x needs nothing else
//        B1x_r[kx <= Nx][yl][z]                                                        (x-stage workspace)
//   forward transpose: rank s receives the kx planes [k0_s, k0_s + np_s) of every rank
//        B1y_s[kxl < np_s][y < Ny][z]                                                  (y-z-stage workspace)
//   K2, K3, K4 work plane by plane -> rank s runs them on its np_s planes with the spectrum rows of those planes
//   backward transpose: back to B1x_r, then K5 along x gives phi_r[x][yl][z].
//
// Every block that moves is a set of `nrun` contiguous runs of run_len = (Ny/P) Nz complex numbers, so the transpose
// is a strided copy written straight into the destination rank's workspace through peer memory (NVLink P2P stores):
// no pack buffer, no unpack pass.  Bytes leaving a GPU per solve: 2 x 16 (Nx+1)(Ny/P) Nz (P-1)/P.
// The index arithmetic lives in shard_planes / shard_block (host functions, exported through the C ABI so that a
// CPU test can push a labelled array through the same numbers).
#pragma once
#include <cuda_runtime.h>

namespace fsp {

constexpr int kMaxRanks = 16;

// kx planes of rank `rank`: the Nx + 1 planes are dealt out in contiguous slabs, the first (Nx+1) % P ranks hold one more
inline void shard_planes(int Nx, int nranks, int rank, int* k0, int* np) {
    const int total = Nx + 1, base = total / nranks, rem = total % nranks;
    *np = base + (rank < rem ? 1 : 0);
    *k0 = rank * base + (rank < rem ? rank : rem);
}

struct ShardBlock { long nrun, run_len, src_off, src_stride, dst_off, dst_stride; };   // in complex (16-byte) elements

// The block rank `src` sends to rank `dst`.
//   direction 0 (forward):  from B1x_src[kx][yl][z]   to B1y_dst[kxl][y][z]   (planes of dst, y-slab of src)
//   direction 1 (backward): from B1y_src[kxl][y][z]   to B1x_dst[kx][yl][z]   (planes of src, y-slab of dst)
inline ShardBlock shard_block(int Nx, int Ny, int Nz, int nranks, int src, int dst, int direction) {
    const long yl = Ny / nranks, run = yl * (long)Nz;
    int k0, np;
    ShardBlock b;
    b.run_len = run;
    if (direction == 0) {
        shard_planes(Nx, nranks, dst, &k0, &np);
        b.nrun = np;
        b.src_off = (long)k0 * run;          b.src_stride = run;
        b.dst_off = (long)src * run;         b.dst_stride = (long)Ny * Nz;
    } else {
        shard_planes(Nx, nranks, src, &k0, &np);
        b.nrun = np;
        b.src_off = (long)dst * run;         b.src_stride = (long)Ny * Nz;
        b.dst_off = (long)k0 * run;          b.dst_stride = run;
    }
    return b;
}

// one launch moves the blocks for all destination ranks: blockIdx.y = destination
struct ShardCopyArgs {
    double2* dst[kMaxRanks];
    ShardBlock blk[kMaxRanks];
};

__global__ void k_shard_copy(const double2* __restrict__ src, const ShardCopyArgs a) {
    const ShardBlock b = a.blk[blockIdx.y];
    double2* __restrict__ dst = a.dst[blockIdx.y];
    const long total = b.nrun * b.run_len;
    for (long e = blockIdx.x * (long)blockDim.x + threadIdx.x; e < total; e += (long)gridDim.x * blockDim.x) {
        const long r = e / b.run_len, i = e - r * b.run_len;
        dst[b.dst_off + r * b.dst_stride + i] = src[b.src_off + r * b.src_stride + i];
    }
}

}  // namespace fsp

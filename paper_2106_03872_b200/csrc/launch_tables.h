// launch_tables.h -- host-side tables of kernel entry points, one row per supported size (16, 32, 48, 64, 96).
#pragma once
#include <cstddef>

namespace tdh {

struct TileLaunch {
    const void* fwd;   // tile_fwd_kernel<NY,NZ,false>
    const void* fwd_slab;  // tile_fwd_kernel<NY,NZ,true>: spectrum rows stored into the ranks' Fourier-space slabs
    const void* inv[5];  // tile_inv_kernel<NY,NZ,CM>, CM = 0 (no projectors), 1, 4, 9, 16 (tile_kernels.cuh, nl_cm_index)
    int threads;
    int ppc;           // plane parts per CTA
    int s;             // y-split: a plane is s parts (rows y = s*m + r)
    int r1y, r2y;      // factorisation of the y transform of length NY/s (row order inside a tile)
    int r1z;           // NZ / 8 (128-byte lines per row)
    size_t smem_fwd;   // dynamic shared memory per CTA of tile_fwd (ring of tiles)
    size_t smem_inv;   // dynamic shared memory per CTA of tile_inv (the same ring)
};

struct XLaunch {
    const void* fused;  // xpencil_kernel<NX,S,0>
    const void* fwd;    // xpencil_kernel<NX,S,1>
    const void* inv;    // xpencil_kernel<NX,S,2>
    const void* poisson;  // xpencil_kernel<NX,S,3>
    const void* teter;    // xpencil_kernel<NX,S,4>
    const void* fused_slab;  // xpencil_kernel<NX,S,0,true>: pencils of a Fourier-space slab, x values stored to their owners
    const void* inv_slab;    // xpencil_kernel<NX,S,2,true>
    int threads;
    size_t smem;        // dynamic shared memory per CTA (ring of tiles)
};

// defined in tile_nz<NZ>.cu / xpencil_inst.cu; return false for an unsupported size
bool tile_launch_nz16(int ny, TileLaunch* out);
bool tile_launch_nz32(int ny, TileLaunch* out);
bool tile_launch_nz48(int ny, TileLaunch* out);
bool tile_launch_nz64(int ny, TileLaunch* out);
bool tile_launch_nz96(int ny, TileLaunch* out);
bool xpencil_launch(int nx, int s, XLaunch* out);

}  // namespace tdh

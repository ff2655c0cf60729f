// launch_tables.h -- host-side tables of kernel entry points, one row per supported size (16, 32, 48, 64, 96).
#pragma once
#include <cstddef>

namespace tdh {

struct PlaneLaunch {
    const void* fwd;   // plane_fwd_kernel<NY,NZ>
    const void* inv;   // plane_inv_kernel<NY,NZ>
    int threads;
    int ppc;           // planes per CTA
    size_t smem;       // dynamic shared memory per CTA
};

struct XLaunch {
    const void* fused;  // xpencil_kernel<NX,0>
    const void* fwd;    // xpencil_kernel<NX,1>
    const void* inv;    // xpencil_kernel<NX,2>
    int threads;
};

// defined in plane_nz<NZ>.cu / xpencil_inst.cu; return false for an unsupported size
bool plane_launch_nz16(int ny, PlaneLaunch* out);
bool plane_launch_nz32(int ny, PlaneLaunch* out);
bool plane_launch_nz48(int ny, PlaneLaunch* out);
bool plane_launch_nz64(int ny, PlaneLaunch* out);
bool plane_launch_nz96(int ny, PlaneLaunch* out);
bool xpencil_launch(int nx, XLaunch* out);

}  // namespace tdh

// xpencil_inst.cu -- instantiates the x-pencil kernels for every supported NX and both y-splits.
#include "xpencil_kernel.cuh"
#include "launch_tables.h"

namespace tdh {

template <int NX, int S> static XLaunch make_x_launch() {
    XLaunch x;
    x.fused = reinterpret_cast<const void*>(&xpencil_kernel<NX, S, 0>);
    x.fwd = reinterpret_cast<const void*>(&xpencil_kernel<NX, S, 1>);
    x.inv = reinterpret_cast<const void*>(&xpencil_kernel<NX, S, 2>);
    x.poisson = reinterpret_cast<const void*>(&xpencil_kernel<NX, S, 3>);
    x.teter = reinterpret_cast<const void*>(&xpencil_kernel<NX, S, 4>);
    x.fused_slab = reinterpret_cast<const void*>(&xpencil_kernel<NX, S, 0, true>);
    x.inv_slab = reinterpret_cast<const void*>(&xpencil_kernel<NX, S, 2, true>);
    x.threads = XCfg<NX>::T;
    x.smem = XCfg<NX>::SMEM;
    return x;
}

template <int S> static bool x_launch_s(int nx, XLaunch* out) {
    switch (nx) {
        case 16: *out = make_x_launch<16, S>(); return true;
        case 32: *out = make_x_launch<32, S>(); return true;
        case 48: *out = make_x_launch<48, S>(); return true;
        case 64: *out = make_x_launch<64, S>(); return true;
        case 96: *out = make_x_launch<96, S>(); return true;
        default: return false;
    }
}

bool xpencil_launch(int nx, int s, XLaunch* out) {
    if (s == 1) return x_launch_s<1>(nx, out);
    if (s == 2) return x_launch_s<2>(nx, out);
    return false;
}

}  // namespace tdh

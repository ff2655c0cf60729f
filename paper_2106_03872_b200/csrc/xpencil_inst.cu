// xpencil_inst.cu -- instantiates the x-pencil kernels for every supported NX.
#include "fft_kernels.cuh"
#include "launch_tables.h"

namespace tdh {

template <int NX> static XLaunch make_x_launch() {
    XLaunch x;
    x.fused = reinterpret_cast<const void*>(&xpencil_kernel<NX, 0>);
    x.fwd = reinterpret_cast<const void*>(&xpencil_kernel<NX, 1>);
    x.inv = reinterpret_cast<const void*>(&xpencil_kernel<NX, 2>);
    x.threads = XP_LPC * Fact<NX>::R1;
    return x;
}

bool xpencil_launch(int nx, XLaunch* out) {
    switch (nx) {
        case 16: *out = make_x_launch<16>(); return true;
        case 32: *out = make_x_launch<32>(); return true;
        case 48: *out = make_x_launch<48>(); return true;
        case 64: *out = make_x_launch<64>(); return true;
        case 96: *out = make_x_launch<96>(); return true;
        default: return false;
    }
}

}  // namespace tdh

// peak_probe.cu -- measurement of the FP64 tensor-core (DMMA) issue ceiling of the device, for the roofline denominators
// of the contraction kernels ("a dependent-free mma.sync f64 issue loop").  Not part of the
// product library or its ABI: built into its own libtdh_probe.so (paper_2106_03872_b200/build.py), which only bench.py
// loads; it reports the figure beside the cuBLAS DGEMM rate measured in the same run.
#include <cuda_runtime.h>

namespace {

constexpr int NACC = 8;        // independent accumulator chains per warp
constexpr int UNROLL = 8;

__global__ void __launch_bounds__(256) dmma_issue_kernel(double* sink, int iters, double a0, double b0) {
    double c[NACC][2];
#pragma unroll
    for (int i = 0; i < NACC; ++i) c[i][0] = c[i][1] = 0.0;
    const double a = a0 + 1e-9 * threadIdx.x, b = b0 - 1e-9 * threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
#pragma unroll
            for (int i = 0; i < NACC; ++i)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                             : "+d"(c[i][0]), "+d"(c[i][1])
                             : "d"(a), "d"(b));
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < NACC; ++i) s += c[i][0] + c[i][1];
    if (s == 123.456) sink[0] = s;          // keeps the chains alive
}

}  // namespace

// FP64 tensor-core issue ceiling in TFLOP/s: every warp of a full grid (all SMs, 8 warps x as many CTAs as fit) issues
// independent mma.sync.m8n8k4.f64 instructions (512 flop each) from registers; best of three timed launches.
// returns 0, or -1 bad argument / -3 allocation failed / -4 CUDA error
extern "C" int probe_fp64_mma_peak(double* tflops_out) {
    if (!tflops_out) return -1;
    int dev = 0, nsm = 0, occ = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -4;
    if (cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -4;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, dmma_issue_kernel, 256, 0) != cudaSuccess || occ < 1) return -4;
    double* sink = nullptr;
    if (cudaMalloc(&sink, sizeof(double)) != cudaSuccess) return -3;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int ctas = nsm * occ, iters = 4096;
    double best = 0.0;
    int rc = 0;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, 0);
        dmma_issue_kernel<<<ctas, 256>>>(sink, iters, 1.0, 0.5);
        cudaEventRecord(e1, 0);
        if (cudaEventSynchronize(e1) != cudaSuccess) { rc = -4; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flops = (double)ctas * 8.0 * (double)iters * UNROLL * NACC * 512.0;
        if (rep > 0 && ms > 0.f) best = flops / (ms * 1e-3) * 1e-12 > best ? flops / (ms * 1e-3) * 1e-12 : best;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    *tflops_out = best;
    return rc;
}

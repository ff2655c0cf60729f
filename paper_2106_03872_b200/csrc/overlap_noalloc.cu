// overlap_noalloc.cu -- tdh_overlap_noalloc (include/tdh.h): the overlap matrix of two state blocks,
//
//     S[i][j] = dV sum_p conj(a_i[p]) b_j[p],   i < na, j < nb
//
// for callers that are not allowed to allocate device memory.  Who that is: a host program that has handed the whole
// device to its own memory pool (INQ itself keeps a pool so that "no allocation happens on hot paths"; a
// second allocator asking the driver for memory next to such a pool fails or fragments it), a time-stepping loop that
// cannot afford cudaMalloc's implicit device-wide synchronisation in the middle of its asynchronous work, and code that
// gets no handle at all: a tdh_grid allocates gigabytes of workspace when it is created, which is too much to ask of
// somebody who only wants to check that a small block of states is still orthonormal.
//
// tdh_overlap keeps the partial tiles of its split-K GEMM in the handle's workspace.  This variant keeps them in ONE
// file-scope device array of fixed size (TDH_NOALLOC_SCRATCH_BYTES = 8 MiB, part of the library image: every device that
// loads libtdh.so holds these 8 MiB until the process exits), needs no handle, and calls neither cudaMalloc nor cudaFree
// nor any library routine that allocates.  The price is a size limit (na, nb <= TDH_NOALLOC_MAX_STATES) and that all
// calls of the process share the array: two calls whose kernels may run at the same time on one device (different
// streams, different host threads) race on it and produce garbage; calls on one stream are ordered and safe.
//
// Nothing in the array has to start at zero: the first kernel of a call writes every cell the second kernel of the same
// call reads (whole 64 x 64 tiles, rows and columns beyond na / nb as zeros from predicated loads), so whatever the
// previous call left behind is overwritten or never looked at.
//
// The array's name is only a host-side stand-in in host code, not a device address.  The first call on a device asks
// the runtime for the real address (cudaGetSymbolAddress, with that device current) and remembers it per device; the
// kernels get that pointer as an argument.  That first call also makes the runtime load this module on the device, so
// it should be made once at start-up, before the caller begins a stream capture or enters the part of its program
// where it must not block.
//
// The kernels are the ones of overlap_kernels.cuh (64 x 64 tile of S per CTA, one slice of K per grid row, chunks of 16
// points through padded shared-memory planes, mma.sync.m8n8k4.f64) restated here with one difference: the last chunk
// of K is predicated, so the number of points needs no particular divisibility.  The existing path is untouched.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cstdio>
#include <mutex>

#include "../../include/tdh.h"

int tdh_detail_set_error(int code, const char* msg);      // tdh.cu: stores the text tdh_last_error() returns

namespace {

typedef double2 cd;

constexpr int NA_T = 64;           // tile edge (states)
constexpr int NA_KC = 16;          // points per chunk
constexpr int NA_KCP = 20;         // padded row length (doubles): fragment reads fall into 32 distinct banks
constexpr int NA_THREADS = 256;
constexpr size_t NA_CELLS = (size_t)TDH_NOALLOC_SCRATCH_BYTES / sizeof(cd);
constexpr int NA_MAX_DEVICES = 64;

// The scratch: [ksplit][na_pad][nb_pad] partial tiles of the current call.  Shared by every call of the process.
static __device__ __align__(256) cd g_noalloc_scratch[NA_CELLS];

__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c[0]), "+d"(c[1])
                 : "d"(a), "d"(b));
}

// grid: (tiles_i * tiles_j, ksplit); slice blockIdx.y covers chunks [y*cps, (y+1)*cps) of the ceil(npts/16) chunks.
// hermitian != 0 (one block against itself): tiles below the diagonal are skipped, the reduction mirrors them.
__global__ void __launch_bounds__(NA_THREADS)
overlap_noalloc_kernel(const cd* __restrict__ a, int na, const cd* __restrict__ b, int nb, size_t npts, int tiles_j,
                       int cps, cd* __restrict__ part, int hermitian)
{
    if (hermitian && (int)(blockIdx.x % tiles_j) < (int)(blockIdx.x / tiles_j)) return;
    __shared__ double sre[2 * NA_T][NA_KCP];     // rows 0..63: states of a, rows 64..127: states of b
    __shared__ double sim[2 * NA_T][NA_KCP];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wi = warp >> 2, wj = warp & 3;                    // warps as 2 x 4, a warp owns 32 x 16 of the tile
    const int fr = lane >> 2, fk = lane & 3;                    // fragment row (state) and k (point)
    const int ti = blockIdx.x / tiles_j, tj = blockIdx.x % tiles_j;
    const int i0 = ti * NA_T, j0 = tj * NA_T;
    const size_t nchunks = (npts + NA_KC - 1) / NA_KC;
    const size_t c_begin = (size_t)blockIdx.y * cps;
    const size_t c_end = c_begin + cps < nchunks ? c_begin + cps : nchunks;

    // load slot r of this thread: row (tid + 256 r) / 16 of the 128-row tile, point (tid + 256 r) % 16 of the chunk
    const cd* src[8];
    bool ok[8];
    const int pt = tid & 15;
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const int row = (tid + NA_THREADS * r) >> 4;
        const bool isb = row >= NA_T;
        const int st = isb ? j0 + row - NA_T : i0 + row;
        ok[r] = isb ? st < nb : st < na;
        src[r] = (isb ? b : a) + (size_t)(ok[r] ? st : 0) * npts + pt;
    }
    double cre[4][2][2], cim[4][2][2];
#pragma unroll
    for (int it = 0; it < 4; ++it)
#pragma unroll
        for (int jt = 0; jt < 2; ++jt) cre[it][jt][0] = cre[it][jt][1] = cim[it][jt][0] = cim[it][jt][1] = 0.0;

    cd v[8];
    auto load = [&](size_t c) {
        const bool inside = c * NA_KC + pt < npts;               // the last chunk may be ragged
#pragma unroll
        for (int r = 0; r < 8; ++r) v[r] = (ok[r] && inside) ? __ldcs(src[r] + c * NA_KC) : make_double2(0.0, 0.0);
    };
    if (c_begin < c_end) load(c_begin);
    for (size_t c = c_begin; c < c_end; ++c) {
        __syncthreads();                                         // the previous chunk has been consumed
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int row = (tid + NA_THREADS * r) >> 4;
            sre[row][pt] = v[r].x;
            sim[row][pt] = v[r].y;
        }
        __syncthreads();
        if (c + 1 < c_end) load(c + 1);                          // in flight during the multiplications below
#pragma unroll
        for (int k4 = 0; k4 < NA_KC / 4; ++k4) {
            double ar[4], ai[4], br[2], bi[2];
#pragma unroll
            for (int it = 0; it < 4; ++it) {
                ar[it] = sre[wi * 32 + it * 8 + fr][k4 * 4 + fk];
                ai[it] = sim[wi * 32 + it * 8 + fr][k4 * 4 + fk];
            }
#pragma unroll
            for (int jt = 0; jt < 2; ++jt) {
                br[jt] = sre[NA_T + wj * 16 + jt * 8 + fr][k4 * 4 + fk];
                bi[jt] = sim[NA_T + wj * 16 + jt * 8 + fr][k4 * 4 + fk];
            }
#pragma unroll
            for (int it = 0; it < 4; ++it)
#pragma unroll
                for (int jt = 0; jt < 2; ++jt) {                 // conj(a) b = (ar br + ai bi) + i (ar bi - ai br)
                    dmma(cre[it][jt], ar[it], br[jt]);
                    dmma(cre[it][jt], ai[it], bi[jt]);
                    dmma(cim[it][jt], ar[it], bi[jt]);
                    dmma(cim[it][jt], -ai[it], br[jt]);
                }
        }
    }
    // C fragment: row = lane/4, columns 2*(lane%4) + {0,1}.  The whole tile is written, zeros included.
    const int nb_pad = tiles_j * NA_T;
    const size_t na_pad = (size_t)gridDim.x / tiles_j * NA_T;
    cd* dst = part + (size_t)blockIdx.y * na_pad * nb_pad;
#pragma unroll
    for (int it = 0; it < 4; ++it)
#pragma unroll
        for (int jt = 0; jt < 2; ++jt) {
            const int i = i0 + wi * 32 + it * 8 + fr, j = j0 + wj * 16 + jt * 8 + 2 * fk;
            dst[(size_t)i * nb_pad + j] = make_double2(cre[it][jt][0], cim[it][jt][0]);
            dst[(size_t)i * nb_pad + j + 1] = make_double2(cre[it][jt][1], cim[it][jt][1]);
        }
}

// s[i][j] = dv * (sum over the slices, in slice order, of part[ks][i][j]); with hermitian set, an element in a tile below
// the diagonal is the conjugate of its mirror image
__global__ void overlap_noalloc_reduce_kernel(const cd* __restrict__ part, int ksplit, int na, int nb, int na_pad,
                                              int nb_pad, double dv, cd* __restrict__ s, int hermitian)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= na * nb) return;
    int i = idx / nb, j = idx % nb;
    const bool mirror = hermitian && (j / NA_T) < (i / NA_T);
    if (mirror) { const int t = i; i = j; j = t; }
    double re = 0.0, im = 0.0;
    for (int ks = 0; ks < ksplit; ++ks) {
        const cd v = part[((size_t)ks * na_pad + i) * nb_pad + j];
        re += v.x;
        im += v.y;
    }
    s[idx] = make_double2(dv * re, mirror ? -dv * im : dv * im);
}

// Per device: the device address of g_noalloc_scratch and the SM count, looked up once, with that device current.
struct DeviceSetup { std::atomic<cd*> scratch{nullptr}; int nsm = 0; };
DeviceSetup g_setup[NA_MAX_DEVICES];
std::mutex g_setup_mutex;

int fail(int code, const char* what, cudaError_t e) {
    char msg[384];
    snprintf(msg, sizeof(msg), "tdh_overlap_noalloc: %s: %s", what, cudaGetErrorString(e));
    return tdh_detail_set_error(code, msg);
}

// Returns the scratch address valid on the CURRENT device (set-up on the first call for that device).
int device_setup(cd** scratch, int* nsm) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(TDH_ECUDA, "cudaGetDevice", e);
    if (dev < 0 || dev >= NA_MAX_DEVICES)
        return tdh_detail_set_error(TDH_EUNSUPPORTED, "tdh_overlap_noalloc: device ordinal beyond 63");
    DeviceSetup& d = g_setup[dev];
    cd* p = d.scratch.load(std::memory_order_acquire);
    if (p == nullptr) {
        std::lock_guard<std::mutex> lock(g_setup_mutex);
        p = d.scratch.load(std::memory_order_relaxed);
        if (p == nullptr) {
            // g_noalloc_scratch in host code names a host-side shadow symbol; this is its address on device `dev`
            void* sym = nullptr;
            e = cudaGetSymbolAddress(&sym, g_noalloc_scratch);
            if (e != cudaSuccess) return fail(TDH_ECUDA, "cudaGetSymbolAddress(scratch)", e);
            if (sym == nullptr) return tdh_detail_set_error(TDH_ECUDA, "tdh_overlap_noalloc: the scratch symbol has no device address");
            e = cudaDeviceGetAttribute(&d.nsm, cudaDevAttrMultiProcessorCount, dev);
            if (e != cudaSuccess) return fail(TDH_ECUDA, "cudaDeviceGetAttribute(SM count)", e);
            p = static_cast<cd*>(sym);
            d.scratch.store(p, std::memory_order_release);
        }
    }
    *scratch = p;
    *nsm = d.nsm;
    return TDH_OK;
}

}  // namespace

extern "C" int tdh_overlap_noalloc(size_t npts, double dv, int na, const tdh_c128* a_dev, int nb, const tdh_c128* b_dev,
                                   tdh_c128* s_dev, void* cuda_stream) {
    if (!a_dev || !b_dev || !s_dev) return tdh_detail_set_error(TDH_EINVAL, "tdh_overlap_noalloc: null argument");
    if (na < 1 || nb < 1 || npts < 1) return tdh_detail_set_error(TDH_EINVAL, "tdh_overlap_noalloc: na, nb and npts must be >= 1");
    if (na > TDH_NOALLOC_MAX_STATES || nb > TDH_NOALLOC_MAX_STATES) {
        char msg[256];
        snprintf(msg, sizeof(msg), "tdh_overlap_noalloc: %d x %d states is beyond the %d x %d the fixed %d MiB scratch array is "
                 "laid out for; use tdh_overlap (handle workspace) for larger blocks", na, nb, TDH_NOALLOC_MAX_STATES,
                 TDH_NOALLOC_MAX_STATES, (int)(TDH_NOALLOC_SCRATCH_BYTES >> 20));
        return tdh_detail_set_error(TDH_EUNSUPPORTED, msg);
    }
    cd* part = nullptr;
    int nsm = 0;
    if (int rc = device_setup(&part, &nsm)) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);

    const int ti = (na + NA_T - 1) / NA_T, tj = (nb + NA_T - 1) / NA_T;
    const size_t tile_cells = (size_t)ti * tj * NA_T * NA_T;            // <= 65536 cells = 1 MiB per slice of K
    const size_t nchunks = (npts + NA_KC - 1) / NA_KC;
    // slices of K: about eight CTAs per SM, at least 8 chunks per slice, as many as the array holds
    size_t ksplit = std::max<size_t>(1, ((size_t)8 * nsm + (size_t)ti * tj - 1) / ((size_t)ti * tj));
    ksplit = std::min(ksplit, std::max<size_t>(1, nchunks / 8));
    ksplit = std::min(ksplit, NA_CELLS / tile_cells);
    const int cps = (int)((nchunks + ksplit - 1) / ksplit);
    ksplit = (nchunks + cps - 1) / cps;
    const int hermitian = (na == nb && a_dev == b_dev) ? 1 : 0;

    overlap_noalloc_kernel<<<dim3(ti * tj, (unsigned)ksplit), NA_THREADS, 0, stream>>>(
        reinterpret_cast<const cd*>(a_dev), na, reinterpret_cast<const cd*>(b_dev), nb, npts, tj, cps, part, hermitian);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(TDH_ECUDA, "launch of overlap_noalloc_kernel", e);
    overlap_noalloc_reduce_kernel<<<(na * nb + 255) / 256, 256, 0, stream>>>(
        part, (int)ksplit, na, nb, ti * NA_T, tj * NA_T, dv, reinterpret_cast<cd*>(s_dev), hermitian);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(TDH_ECUDA, "launch of overlap_noalloc_reduce_kernel", e);
    return TDH_OK;
}

// tdh.cu -- C ABI of libtdh.so (include/tdh.h): handle, tables, projector re-indexing, launch orchestration.
//
// One Hamiltonian application on a chunk of states is four launches, plus one per atom colour on split-tile grids:
//     nl_project  (gather + FP64-MMA projection, only with projectors)
//     plane_fwd   (tile_fwd: z,y forward FFT per tile of a (state,x) plane)   in  -> work
//     xpencil     (x forward, 1/2|G+k|^2 scale + mask, x inverse)             work in place
//     plane_inv   (tile_inv: y,z inverse FFT + epilogue alpha*(T+V[+Vnl])phi + y)  work -> out
//     nl_scatter  (FP64-MMA back-projection added into out by bulk reduce-add of whole z-runs -- the L2 does the
//                  read-modify-write; nl_mode 1 -- otherwise the back-projection runs inside plane_inv from per-tile
//                  record lists)
// tdh_taylor_pair / tdh_etrs_step (NEXT-1) and tdh_density / tdh_hartree (NEXT-2) are compositions of the same
// launches plus three elementwise kernels.
// The three FFT kernels are persistent (one or several CTAs per SM, as many as fit) and fed by TMA: the host encodes a
// CUtensorMap per launch (tensor_maps.h) and the kernels stream tiles through a shared-memory ring.  `work` holds the
// spectrum in the digit-permuted order the in-place transforms produce (xpencil_kernel.cuh, WORK LAYOUT).
// States are independent, so a block is pushed through this chain chunk by chunk; a chunk is as many
// states as the 4 GiB workspace holds (measured: L2-resident small chunks never win, profiles/r01a_chunk_sweep.md).
// propagate runs ALL steps of one chunk before moving to the next chunk (H is fixed: readings R10, R16), evaluating
// Eq. 8 in Horner form  psi + a1 H(psi + a2 H(psi + a3 H(psi + a4 H psi))),  a_k = -i dt / k,  so that every
// application's epilogue is a single fused axpy and no accumulator is read-modified-written.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/tdh.h"
#include "launch_tables.h"
#include "nl_kernels.cuh"
#include "overlap_kernels.cuh"
#include "eigh_kernels.cuh"
#include "tensor_maps.h"
#include "tile_kernels.cuh"
#include "xpencil_kernel.cuh"
#include "generic_fft.cuh"
#include "small_kernels.cuh"

using tdh::cd;

// ------------------------------------------------------------------------------------------------------------
// errors
// ------------------------------------------------------------------------------------------------------------
static thread_local char g_err[512] = "";

static int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CU(call)                                                                                          \
    do {                                                                                                  \
        cudaError_t e_ = (call);                                                                          \
        if (e_ != cudaSuccess)                                                                            \
            return fail(e_ == cudaErrorMemoryAllocation ? TDH_ENOMEM : TDH_ECUDA, "%s: %s (%s:%d)", #call, \
                        cudaGetErrorString(e_), __FILE__, __LINE__);                                      \
    } while (0)

extern "C" const char* tdh_last_error(void) { return g_err; }

// for the other translation units of the library (overlap_noalloc.cu): record the message of a failing call
int tdh_detail_set_error(int code, const char* msg) { return fail(code, "%s", msg); }

// ------------------------------------------------------------------------------------------------------------
// handle
// ------------------------------------------------------------------------------------------------------------
enum { K_NLPROJ = 0, K_PLANE_FWD = 1, K_XPENCIL = 2, K_PLANE_INV = 3, K_NLSCATTER = 4, K_SMALL_H = 5 };
static const char* const kKernelNames[TDH_NKERNELS] = {"nl_project", "plane_fwd", "xpencil", "plane_inv", "nl_scatter",
                                                       "small_h"};

struct ProfRec { cudaEvent_t a, b; int k; };

struct tdh_grid {
    int n[3];
    double len[3], kpt[3], ecut;
    int max_states;
    cudaStream_t stream;
    size_t np;
    double dv;
    bool have_k;

    double* d_v;          // V(r); zero-filled until set
    bool have_v;
    double* d_g2[3];      // (G_a + k_a)^2
    cd* d_tw[3];          // exp(+2 pi i m / N_a)
    double* d_g2y_w;      // (G_y + k_y)^2 per plane row of the work layout
    double* d_g2z_w;      // (G_z + k_z)^2 per column of the work layout
    cd* d_twy_w;          // exp(+2 pi i k / NY) per row pair of the work layout (y-split grids)
    int* d_rowmap;        // natural ky -> plane row of the work layout
    int* d_colmap;        // natural kz -> column of the work layout
    double* d_p2x;        // |G_x|^2 (no Bloch vector): Poisson solver, natural x order
    double* d_p2y_w;      // |G_y|^2, work-layout order
    double* d_p2z_w;      // |G_z|^2, work-layout order
    double* d_occ;        // [max_states] occupations of the last tdh_density call
    double* d_gs[3];      // signed G_a + k_a: x in natural order, y and z in work-layout order (gradient, forces)
    double* d_dvscale;    // [nchan_tot] dV: projections without the KB coefficient (forces)
    cd* d_dpig;           // [chunk_cap][nchan_tot] dV <beta|d_a psi> (forces)
    double* d_gd;         // [3][N_p] sum_s f_s 2 Re conj(d_a psi_s) psi_s (forces, local term)
    double* d_force;      // [natoms][3] + reduction scratch (forces)
    cd* d_small[3];       // n x n scratch of tdh_orthonormalize ([0] overlap / Cholesky factor, [2] rotation), grown on demand
    int small_n;
    int* d_status;        // Cholesky status word
    unsigned* d_ctl;      // tdh_subspace_diag: barrier counter, sweep maximum, sweeps used
    int jacobi_sweeps;    // sweeps of the last tdh_subspace_diag call that returned its eigenvalues
    double* d_w;          // tdh_subspace_diag: eigenvalues
    double* d_sd;         // tdh_sd_step: [max_states] eps, [max_states] T, [max_states * 3 * SD_SLICES] partial sums
    int ctas_fwd, ctas_inv[tdh::NL_NCM], ctas_x[5];   // persistent grid sizes (SM count x resident CTAs)
    int ctas_fwd_slab, ctas_x_slab[2];

    // whole state on chip (small_kernels.cuh): 16^3 (one CTA per state) and 32^3 (a cluster of four CTAs per state)
    int small_cs;         // 0: not available; else the cluster size
    const void* small_fn;
    int small_cells;
    bool small16_cluster; // 16^3: the four-CTA cluster variant for blocks of few states (TDH_SMALL16_CLUSTER=0 switches it off)

    // general axis lengths (generic_fft.cuh): any n[a] = 2^a 3^b in [4, 256] outside the tuned set {16, 32, 48, 64, 96}
    bool generic;
    tdh::GAxis gax[3];    // z, y, x transforms (index = axis)
    int nsm;

    // slab decomposition (tdh_create_slab_grid): n[0] is then the number of LOCAL planes, nx_fs the full NX
    int nx_fs;            // planes the x transform spans (= n[0] unless this is a slab handle)
    size_t np_total;      // grid points of the whole grid
    int slab_world, slab_rank, ny_local;
    cd* d_fs;             // Fourier-space slab [chunk][NX][ny_local][NZ]: target of the ranks' tile_fwd stores
    cd* d_dpi_part;       // this rank's partial projections (summed over the ranks into d_dpi)
    cd* peer_fs[tdh::SLAB_MAX_WORLD];
    cd* peer_rs[tdh::SLAB_MAX_WORLD];
    const cd* peer_dpi[tdh::SLAB_MAX_WORLD];
    bool have_peers;

    int chunk_cap;        // states the workspace can hold
    size_t work_cells;    // complex values d_work holds (>= chunk_cap * np)
    int chunk;            // states pushed through the chain together
    cd* d_work;
    cd* d_phi[2];

    tdh::TileLaunch tl;
    tdh::XLaunch xl;

    // projectors
    int natoms, nchan_tot, mt;
    tdh::AtomDesc* d_atoms;
    int* d_sidx;
    double* d_sbeta;
    cd* d_sphase;
    double* d_dscale;
    cd* d_dpi;
    // back-projection records, grouped by tile (x, r) and layer (tile_kernels.cuh, struct Epilogue)
    int* d_nl_off;
    unsigned* d_nl_cc;
    double* d_nl_beta;
    cd* d_nl_phase;
    int nl_layers, nl_nrec, nl_cmax;
    // separate back-projection kernel: atoms grouped by colour (spheres of one colour share no grid point)
    int nl_mode;                       // 1: nl_scatter kernel per colour after plane_inv; 0: records inside plane_inv
    tdh::AtomDesc* d_atoms_col;        // atoms sorted by colour
    tdh::ScRun* d_sc_runs;             // z-runs of every sphere (nl_scatter_bulk_kernel)
    tdh::ScChunk* d_sc_chunks;         // chunks of runs, per atom (AtomDesc::sc0, scn)
    bool scatter_bulk;                 // back-projection by bulk reduce-add (long z-runs) or by the read-modify-write kernel
                                       // (short runs: one TMA operation per run costs more than it saves); TDH_SCATTER_BULK=0/1
    std::vector<int> col_off;          // [ncolours + 1] offsets into d_atoms_col
    int kt;                            // 4-channel tiles of the back-projection MMA

    // host-buffer path
    int host_chunk;
    cd* d_hin[2];
    cd* d_hout[2];
    cudaStream_t s_h2d, s_d2h;
    cudaEvent_t ev_in[2], ev_k[2], ev_out[2];

    // tdh_propagate on small blocks: the launches of one call captured once into a CUDA graph and replayed while the
    // call's arguments and the handle's tables stay the same (`epoch` counts every change of the handle)
    struct PropGraph { cudaGraphExec_t exec; const void* psi; int nst, nsteps, launches; double dt; unsigned epoch; };
    PropGraph pg[4];      // a few entries: callers that alternate between buffers keep their graphs
    int pg_next;          // round-robin replacement
    unsigned epoch;
    bool use_graph;
    cudaStream_t s_cap;

    // statistics
    int launch_count;
    bool profiling;
    std::vector<ProfRec> prof_pool;
    size_t prof_used;
    double ksec[TDH_NKERNELS];
};

static int size_index(int n) {
    switch (n) {
        case 16: return 0;
        case 32: return 1;
        case 48: return 2;
        case 64: return 3;
        case 96: return 4;
        default: return -1;
    }
}

// frequency index of array index a (numpy fftfreq convention; reading R7)
static int freq_index(int a, int n) {
    if (n % 2 == 0) return a < n / 2 ? a : a - n;
    return a <= (n - 1) / 2 ? a : a - n;
}

static void free_projectors(tdh_grid* g) {
    cudaFree(g->d_atoms); cudaFree(g->d_sidx); cudaFree(g->d_sbeta); cudaFree(g->d_sphase); cudaFree(g->d_dscale);
    cudaFree(g->d_atoms_col); g->d_atoms_col = nullptr; g->col_off.clear();
    cudaFree(g->d_sc_runs); g->d_sc_runs = nullptr; cudaFree(g->d_sc_chunks); g->d_sc_chunks = nullptr;
    cudaFree(g->d_dvscale); g->d_dvscale = nullptr; cudaFree(g->d_dpig); g->d_dpig = nullptr;
    cudaFree(g->d_force); g->d_force = nullptr;
    cudaFree(g->d_dpi); cudaFree(g->d_dpi_part); g->d_dpi_part = nullptr; cudaFree(g->d_nl_off); cudaFree(g->d_nl_cc); cudaFree(g->d_nl_beta); cudaFree(g->d_nl_phase);
    g->d_atoms = nullptr; g->d_sidx = nullptr; g->d_sbeta = nullptr; g->d_sphase = nullptr; g->d_dscale = nullptr;
    g->d_dpi = nullptr; g->d_nl_off = nullptr; g->d_nl_cc = nullptr; g->d_nl_beta = nullptr; g->d_nl_phase = nullptr;
    g->natoms = 0; g->nchan_tot = 0; g->mt = 1;
    g->nl_layers = 0; g->nl_nrec = 0; g->nl_cmax = 0;
}

// Largest number of states one launch may cover: what the workspace holds.  (Rounds 1-2 also bounded launches of the
// small multi-plane tile configurations to 128 MB because tile_fwd failed now and then above that; the cause was a
// phase-parity race in the tile ring, fixed by the armed flags of tile_kernels.cuh -- DESIGN.md section 16.)
static int max_chunk(const tdh_grid* g) { return g->chunk_cap; }

static int default_chunk(const tdh_grid* g) {
    // Measured on B200 (profiles/r01a_chunk_sweep.md): every kernel gets faster with more states per launch and the
    // L2-resident small-chunk variant never wins, so the default is the largest chunk the workspace holds.
    // When a block has to be split anyway: a multiple of 8 states (the N of the projector MMAs), so that no state group
    // of the non-local kernels is ragged.
    const int cap = max_chunk(g);
    int c = (cap < g->max_states && cap >= 8) ? cap / 8 * 8 : cap;
    if (const char* e = getenv("TDH_CHUNK_STATES")) { int v = atoi(e); if (v > 0) c = v; }
    return std::max(1, std::min(c, cap));
}

// n: the FULL grid.  world = 1: an ordinary handle.  world > 1: the handle of rank `rank` of a slab decomposition, which
// owns planes rank * n[0]/world .. of every state in real space and rows rank * n[1]/world .. in Fourier space.
static int create_impl(const int n[3], const double len[3], const double kpt[3], double ecut, int max_states,
                       void* cuda_stream, int rank, int world, tdh_grid** out) {
    if (!n || !len || !kpt || !out) return fail(TDH_EINVAL, "tdh_create_grid: null argument");
    if (max_states < 1) return fail(TDH_EINVAL, "tdh_create_grid: max_states must be >= 1");
    for (int a = 0; a < 3; ++a) {
        if (!(len[a] > 0.0) || !std::isfinite(len[a])) return fail(TDH_EINVAL, "tdh_create_grid: len[%d] must be > 0", a);
        if (!std::isfinite(kpt[a])) return fail(TDH_EINVAL, "tdh_create_grid: kpt[%d] not finite", a);
        tdh::GAxis probe;
        if (!tdh::gfft_factor(n[a], &probe))
            return fail(TDH_EUNSUPPORTED, "tdh_create_grid: n[%d] = %d unsupported (every axis length must be 2^a 3^b in [4, 256])", a, n[a]);
    }
    const bool generic = size_index(n[0]) < 0 || size_index(n[1]) < 0 || size_index(n[2]) < 0;
    if (generic && world > 1)
        return fail(TDH_EUNSUPPORTED, "tdh_create_slab_grid: slab handles exist for axis lengths 16, 32, 48, 64, 96 only");
    if (world < 1 || world > tdh::SLAB_MAX_WORLD || rank < 0 || rank >= world)
        return fail(TDH_EINVAL, "tdh_create_slab_grid: rank %d / world %d (world <= %d)", rank, world, tdh::SLAB_MAX_WORLD);
    if (world > 1 && (n[0] % world != 0 || n[1] % (2 * world) != 0))
        return fail(TDH_EUNSUPPORTED, "tdh_create_slab_grid: world = %d must divide n[0] = %d and n[1] / 2 = %d", world, n[0], n[1] / 2);
    int ndev = 0;
    CU(cudaGetDeviceCount(&ndev));
    if (ndev < 1) return fail(TDH_ECUDA, "tdh_create_grid: no CUDA device (there is no CPU fallback)");

    tdh_grid* g = new (std::nothrow) tdh_grid();
    if (!g) return fail(TDH_ENOMEM, "tdh_create_grid: host allocation failed");
    for (int a = 0; a < 3; ++a) { g->n[a] = n[a]; g->len[a] = len[a]; g->kpt[a] = kpt[a]; }
    g->nx_fs = n[0];
    g->n[0] = n[0] / world;                                   // local planes
    g->slab_world = world;
    g->slab_rank = rank;
    g->ny_local = n[1] / world;
    g->ecut = (ecut > 0.0 && std::isfinite(ecut)) ? ecut : -1.0;
    g->max_states = max_states;
    g->stream = (cudaStream_t)cuda_stream;
    g->np_total = (size_t)n[0] * n[1] * n[2];
    g->np = g->np_total / world;
    g->dv = (len[0] / n[0]) * (len[1] / n[1]) * (len[2] / n[2]);
    g->have_k = kpt[0] != 0.0 || kpt[1] != 0.0 || kpt[2] != 0.0;
    g->mt = 1;

    g->generic = generic;
    for (int a = 0; a < 3; ++a) tdh::gfft_factor(n[a], &g->gax[a]);
    bool ok = generic;
    if (generic) {                              // no tiles: whole planes, natural order (identity work layout)
        memset(&g->tl, 0, sizeof(g->tl));
        memset(&g->xl, 0, sizeof(g->xl));
        g->tl.s = 1; g->tl.ppc = 1; g->tl.r1y = 1; g->tl.r2y = n[1]; g->tl.r1z = 1;
    }
    if (!generic) switch (n[2]) {
        case 16: ok = tdh::tile_launch_nz16(n[1], &g->tl); break;
        case 32: ok = tdh::tile_launch_nz32(n[1], &g->tl); break;
        case 48: ok = tdh::tile_launch_nz48(n[1], &g->tl); break;
        case 64: ok = tdh::tile_launch_nz64(n[1], &g->tl); break;
        case 96: ok = tdh::tile_launch_nz96(n[1], &g->tl); break;
    }
    ok = ok && (generic || tdh::xpencil_launch(n[0], g->tl.s, &g->xl));
    if (!ok) { delete g; return fail(TDH_EUNSUPPORTED, "tdh_create_grid: no kernel for this grid"); }
    if (world > 1 && g->n[0] % g->tl.ppc != 0) {
        const int ppc = g->tl.ppc;
        delete g;
        return fail(TDH_EUNSUPPORTED, "tdh_create_slab_grid: %d local planes are not a multiple of the %d planes of a tile", n[0] / world, ppc);
    }

    int rc = TDH_OK;
    auto body = [&]() -> int {
        int dev = 0, nsm = 0;
        CU(cudaGetDevice(&dev));
        CU(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
        g->nsm = nsm;
        if (generic) {
            size_t smx = 0;
            for (int a = 0; a < 3; ++a) smx = std::max(smx, tdh::gfft_smem(g->gax[a]));
            const void* gf[] = {(const void*)&tdh::gfft_axis_kernel<-1, -1>, (const void*)&tdh::gfft_axis_kernel<+1, -1>,
                                (const void*)&tdh::gfft_axis_kernel<-1, 0>, (const void*)&tdh::gfft_axis_kernel<-1, 1>,
                                (const void*)&tdh::gfft_axis_kernel<-1, 2>, (const void*)&tdh::gfft_axis_kernel<-1, 3>,
                                (const void*)&tdh::gfft_axis_kernel<-1, 4>, (const void*)&tdh::gfft_zinv_epilogue_kernel};
            for (const void* f : gf) CU(cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smx));
        }
        if (!generic && !tdh::encode_tiled_fn()) return fail(TDH_ECUDA, "tdh_create_grid: cuTensorMapEncodeTiled not available from the driver");
        // persistent grids: SM count x the number of CTAs of each kernel that fit on one SM
        constexpr int NK = 9 + tdh::NL_NCM;
        const void* fs[NK] = {g->tl.fwd, g->xl.fused, g->xl.fwd, g->xl.inv, g->xl.poisson, g->xl.teter,
                              g->tl.fwd_slab, g->xl.fused_slab, g->xl.inv_slab};
        size_t sm[NK] = {g->tl.smem_fwd, g->xl.smem, g->xl.smem, g->xl.smem, g->xl.smem, g->xl.smem,
                         g->tl.smem_fwd, g->xl.smem, g->xl.smem};
        int th[NK] = {g->tl.threads, g->xl.threads, g->xl.threads, g->xl.threads, g->xl.threads, g->xl.threads,
                      g->tl.threads, g->xl.threads, g->xl.threads};
        for (int i = 0; i < tdh::NL_NCM; ++i) { fs[9 + i] = g->tl.inv[i]; sm[9 + i] = g->tl.smem_inv; th[9 + i] = g->tl.threads; }
        int ctas[NK];
        for (int i = 0; i < NK; ++i) {
            if (generic) { ctas[i] = 0; continue; }
            if (world == 1 && i >= 6 && i < 9) { ctas[i] = 0; continue; }       // slab kernels: slab handles only
            CU(cudaFuncSetAttribute(fs[i], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm[i]));
            CU(cudaFuncSetAttribute(fs[i], cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared));
            int occ = 0;
            CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fs[i], th[i], sm[i]));
            if (occ < 1) return fail(TDH_ECUDA, "tdh_create_grid: kernel %d does not fit on an SM", i);
            if (const char* e = getenv("TDH_MAX_CTAS_PER_SM")) { int v = atoi(e); if (v > 0) occ = std::min(occ, v); }
            ctas[i] = nsm * occ;
        }
        g->ctas_fwd = ctas[0];
        g->ctas_x[0] = ctas[1]; g->ctas_x[1] = ctas[2]; g->ctas_x[2] = ctas[3]; g->ctas_x[3] = ctas[4]; g->ctas_x[4] = ctas[5];
        for (int i = 0; i < tdh::NL_NCM; ++i) g->ctas_inv[i] = ctas[9 + i];
        g->ctas_fwd_slab = ctas[6]; g->ctas_x_slab[0] = ctas[7]; g->ctas_x_slab[1] = ctas[8];
        {
            const void* fb[4] = {(const void*)&tdh::nl_scatter_bulk_kernel<1>, (const void*)&tdh::nl_scatter_bulk_kernel<2>,
                                 (const void*)&tdh::nl_scatter_bulk_kernel<3>, (const void*)&tdh::nl_scatter_bulk_kernel<4>};
            for (const void* f : fb) CU(cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tdh::SC_SMEM));
            g->scatter_bulk = true;                     // decided per projector table in tdh_set_projectors
        }
        // tables: built on the host exactly as the oracle builds its G vectors (two_pi * m / L + k, then squared)
        const double two_pi = 6.283185307179586476925286766559;
        for (int a = 0; a < 3; ++a) {
            std::vector<double> g2(n[a]);
            std::vector<cd> tw(n[a]);
            for (int i = 0; i < n[a]; ++i) {
                const double ga = two_pi * freq_index(i, n[a]) / len[a] + kpt[a];
                g2[i] = ga * ga;
                const long double ang = 6.283185307179586476925286766559005768L * (long double)i / (long double)n[a];
                tw[i] = make_double2((double)cosl(ang), (double)sinl(ang));
            }
            CU(cudaMalloc(&g->d_g2[a], sizeof(double) * n[a]));
            CU(cudaMalloc(&g->d_tw[a], sizeof(cd) * n[a]));
            CU(cudaMemcpy(g->d_g2[a], g2.data(), sizeof(double) * n[a], cudaMemcpyHostToDevice));
            CU(cudaMemcpy(g->d_tw[a], tw.data(), sizeof(cd) * n[a], cudaMemcpyHostToDevice));
        }
        // the same tables in the order of the work layout (xpencil_kernel.cuh): plane row Y = S*rho + r with
        // rho = k1y*R2Y + k2y <-> k = k1y + R1Y*k2y and ky = k + r*NY/S; column z' = 8*k1 + k2 <-> kz = k1 + (NZ/8)*k2
        {
            const int ny = n[1], nz = n[2], S = g->tl.s, nys = ny / S, r1y = g->tl.r1y, r2y = g->tl.r2y, r1z = g->tl.r1z;
            std::vector<int> rowmap(ny), colmap(nz);
            std::vector<double> g2y_w(ny), g2z_w(nz);
            std::vector<cd> twy_w(ny / 2);
            for (int ky = 0; ky < ny; ++ky) {
                const int h = ky / nys, k = ky % nys;
                const int rho = generic ? k : (k % r1y) * r2y + k / r1y;
                rowmap[ky] = S * rho + h;
                const double ga = two_pi * freq_index(ky, ny) / len[1] + kpt[1];
                g2y_w[rowmap[ky]] = ga * ga;
                if (S == 2 && h == 0) {
                    const long double ang = 6.283185307179586476925286766559005768L * (long double)k / (long double)ny;
                    twy_w[rho] = make_double2((double)cosl(ang), (double)sinl(ang));
                }
            }
            if (S == 1) for (auto& w : twy_w) w = make_double2(1.0, 0.0);
            for (int kz = 0; kz < nz; ++kz) {
                colmap[kz] = generic ? kz : 8 * (kz % r1z) + kz / r1z;
                const double ga = two_pi * freq_index(kz, nz) / len[2] + kpt[2];
                g2z_w[colmap[kz]] = ga * ga;
            }
            CU(cudaMalloc(&g->d_g2y_w, sizeof(double) * ny));
            CU(cudaMalloc(&g->d_g2z_w, sizeof(double) * nz));
            CU(cudaMalloc(&g->d_twy_w, sizeof(cd) * (ny / 2)));
            CU(cudaMalloc(&g->d_rowmap, sizeof(int) * ny));
            CU(cudaMalloc(&g->d_colmap, sizeof(int) * nz));
            CU(cudaMemcpy(g->d_g2y_w, g2y_w.data(), sizeof(double) * ny, cudaMemcpyHostToDevice));
            CU(cudaMemcpy(g->d_g2z_w, g2z_w.data(), sizeof(double) * nz, cudaMemcpyHostToDevice));
            CU(cudaMemcpy(g->d_twy_w, twy_w.data(), sizeof(cd) * (ny / 2), cudaMemcpyHostToDevice));
            CU(cudaMemcpy(g->d_rowmap, rowmap.data(), sizeof(int) * ny, cudaMemcpyHostToDevice));
            CU(cudaMemcpy(g->d_colmap, colmap.data(), sizeof(int) * nz, cudaMemcpyHostToDevice));
            // |G|^2 tables of the Poisson solver (tdh_hartree): the same orders, without the Bloch vector
            std::vector<double> p2x(n[0]), p2y_w(ny), p2z_w(nz);
            for (int kx = 0; kx < n[0]; ++kx) { const double ga = two_pi * freq_index(kx, n[0]) / len[0]; p2x[kx] = ga * ga; }
            for (int ky = 0; ky < ny; ++ky) { const double ga = two_pi * freq_index(ky, ny) / len[1]; p2y_w[rowmap[ky]] = ga * ga; }
            for (int kz = 0; kz < nz; ++kz) { const double ga = two_pi * freq_index(kz, nz) / len[2]; p2z_w[colmap[kz]] = ga * ga; }
            CU(cudaMalloc(&g->d_p2x, sizeof(double) * n[0]));
            CU(cudaMalloc(&g->d_p2y_w, sizeof(double) * ny));
            CU(cudaMalloc(&g->d_p2z_w, sizeof(double) * nz));
            CU(cudaMemcpy(g->d_p2x, p2x.data(), sizeof(double) * n[0], cudaMemcpyHostToDevice));
            CU(cudaMemcpy(g->d_p2y_w, p2y_w.data(), sizeof(double) * ny, cudaMemcpyHostToDevice));
            CU(cudaMemcpy(g->d_p2z_w, p2z_w.data(), sizeof(double) * nz, cudaMemcpyHostToDevice));
            CU(cudaMalloc(&g->d_occ, sizeof(double) * max_states));
            // signed G_a + k_a (gradient): x natural, y and z in work-layout order
            std::vector<double> gsx(n[0]), gsy(ny), gsz(nz);
            for (int kx = 0; kx < n[0]; ++kx) gsx[kx] = two_pi * freq_index(kx, n[0]) / len[0] + kpt[0];
            for (int ky = 0; ky < ny; ++ky) gsy[rowmap[ky]] = two_pi * freq_index(ky, ny) / len[1] + kpt[1];
            for (int kz = 0; kz < nz; ++kz) gsz[colmap[kz]] = two_pi * freq_index(kz, nz) / len[2] + kpt[2];
            const std::vector<double>* gsv[3] = {&gsx, &gsy, &gsz};
            for (int a = 0; a < 3; ++a) {
                CU(cudaMalloc(&g->d_gs[a], sizeof(double) * n[a]));
                CU(cudaMemcpy(g->d_gs[a], gsv[a]->data(), sizeof(double) * n[a], cudaMemcpyHostToDevice));
            }
        }
        // one-launch path for the grids whose state fits on chip (TDH_SMALL=0 switches it off: the tests run both paths)
        g->small_cs = 0;
        if (!generic && world == 1 && n[0] == n[1] && n[1] == n[2] && (n[0] == 16 || n[0] == 32)) {
            const char* e = getenv("TDH_SMALL");
            if (!(e && atoi(e) == 0)) {
                if (n[0] == 16) { g->small_cs = 1; g->small_fn = (const void*)&tdh::small_h_kernel<16, 1>; g->small_cells = tdh::SmallCfg<16, 1>::CELLS; }
                else { g->small_cs = 4; g->small_fn = (const void*)&tdh::small_h_kernel<32, 4>; g->small_cells = tdh::SmallCfg<32, 4>::CELLS; }
                g->small16_cluster = n[0] == 16;
                if (const char* e2 = getenv("TDH_SMALL16_CLUSTER")) g->small16_cluster = g->small16_cluster && atoi(e2) != 0;
                if (n[0] == 16)
                    CU(cudaFuncSetAttribute((const void*)&tdh::small_h_kernel<16, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            (int)(tdh::SMALL_HEADER + (size_t)tdh::SmallCfg<16, 4>::CELLS * sizeof(cd) +
                                                  (size_t)(tdh::SMALL_SEG_ENTRIES + 2 * tdh::SMALL_MAX_CHAN + 16) * sizeof(cd))));
                CU(cudaFuncSetAttribute(g->small_fn, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        (int)(tdh::SMALL_HEADER + (size_t)g->small_cells * sizeof(cd) +
                                              (size_t)(tdh::SMALL_SEG_ENTRIES + 2 * tdh::SMALL_MAX_CHAN + 16) * sizeof(cd))));
            }
        }
        CU(cudaMalloc(&g->d_v, sizeof(double) * g->np));
        CU(cudaMemset(g->d_v, 0, sizeof(double) * g->np));
        g->have_v = false;
        // workspace: up to 4 GiB per buffer (TDH_WORKSPACE_MB overrides)
        const size_t state_bytes = g->np * sizeof(cd);
        // three block buffers of this size (work, two Horner buffers): 12 GiB of the 180 GB when max_states needs them.
        // Measured on Large (profiles/r01f_summary.md): 1 GiB 26.05 ms per step, 2 GiB 25.88, 4 GiB 25.27 (fewer, longer launches)
        size_t ws_bytes = (size_t)4 << 30;
        if (const char* e = getenv("TDH_WORKSPACE_MB")) { long v = atol(e); if (v > 0) ws_bytes = (size_t)v << 20; }
        size_t cap = std::max<size_t>(1, ws_bytes / state_bytes);
        g->chunk_cap = (int)std::min<size_t>(cap, (size_t)max_states);
        // the work buffer also holds the split-K partial tiles of tdh_overlap: on very small grids (9^3 ...) a chunk of
        // states is smaller than one padded tile grid of the block, so it is at least that (<= 16 MiB)
        {
            const size_t pad = ((size_t)std::min(max_states, 1024) + 63) / 64 * 64;
            g->work_cells = std::max<size_t>((size_t)g->chunk_cap * g->np, pad * pad);
        }
        CU(cudaMalloc(&g->d_work, sizeof(cd) * g->work_cells));
        // at least two states each: tdh_taylor_pair keeps phi_2 and phi_3 in the two halves of d_phi[0]
        CU(cudaMalloc(&g->d_phi[0], state_bytes * std::max(2, g->chunk_cap)));
        CU(cudaMalloc(&g->d_phi[1], state_bytes * std::max(2, g->chunk_cap)));
        if (world > 1) CU(cudaMalloc(&g->d_fs, state_bytes * g->chunk_cap));
        g->chunk = default_chunk(g);
        g->use_graph = true;
        if (const char* e = getenv("TDH_GRAPH")) g->use_graph = atoi(e) != 0;
        return TDH_OK;
    };
    rc = body();
    if (rc != TDH_OK) { tdh_destroy_grid(g); return rc; }
    *out = g;
    return TDH_OK;
}

extern "C" int tdh_create_grid(const int n[3], const double len[3], const double kpt[3], double ecut, int max_states,
                               void* cuda_stream, tdh_grid** out) {
    return create_impl(n, len, kpt, ecut, max_states, cuda_stream, 0, 1, out);
}

extern "C" int tdh_create_slab_grid(const int n[3], const double len[3], const double kpt[3], double ecut, int max_states,
                                    int rank, int world, void* cuda_stream, tdh_grid** out) {
    if (world < 2) return fail(TDH_EINVAL, "tdh_create_slab_grid: world must be >= 2 (tdh_create_grid makes an undivided grid)");
    return create_impl(n, len, kpt, ecut, max_states, cuda_stream, rank, world, out);
}

extern "C" int tdh_destroy_grid(tdh_grid* g) {
    if (!g) return TDH_OK;
    cudaStreamSynchronize(g->stream);
    free_projectors(g);
    cudaFree(g->d_v);
    for (int a = 0; a < 3; ++a) { cudaFree(g->d_g2[a]); cudaFree(g->d_tw[a]); }
    cudaFree(g->d_g2y_w); cudaFree(g->d_g2z_w); cudaFree(g->d_twy_w); cudaFree(g->d_rowmap); cudaFree(g->d_colmap);
    cudaFree(g->d_p2x); cudaFree(g->d_p2y_w); cudaFree(g->d_p2z_w); cudaFree(g->d_occ);
    for (int a = 0; a < 3; ++a) cudaFree(g->d_gs[a]);
    cudaFree(g->d_gd);
    for (int i = 0; i < 3; ++i) cudaFree(g->d_small[i]);
    cudaFree(g->d_status); cudaFree(g->d_sd); cudaFree(g->d_ctl); cudaFree(g->d_w);
    cudaFree(g->d_work); cudaFree(g->d_phi[0]); cudaFree(g->d_phi[1]); cudaFree(g->d_fs);
    for (int i = 0; i < 2; ++i) {
        cudaFree(g->d_hin[i]); cudaFree(g->d_hout[i]);
        if (g->ev_in[i]) cudaEventDestroy(g->ev_in[i]);
        if (g->ev_k[i]) cudaEventDestroy(g->ev_k[i]);
        if (g->ev_out[i]) cudaEventDestroy(g->ev_out[i]);
    }
    for (auto& e : g->pg) if (e.exec) cudaGraphExecDestroy(e.exec);
    if (g->s_cap) cudaStreamDestroy(g->s_cap);
    if (g->s_h2d) cudaStreamDestroy(g->s_h2d);
    if (g->s_d2h) cudaStreamDestroy(g->s_d2h);
    for (auto& r : g->prof_pool) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    delete g;
    return TDH_OK;
}

extern "C" int tdh_set_potential(tdh_grid* g, const double* v_dev) {
    if (!g) return fail(TDH_EINVAL, "tdh_set_potential: null handle");
    g->epoch += 1;
    if (v_dev) {
        CU(cudaMemcpyAsync(g->d_v, v_dev, sizeof(double) * g->np, cudaMemcpyDeviceToDevice, g->stream));
        g->have_v = true;
    } else {
        CU(cudaMemsetAsync(g->d_v, 0, sizeof(double) * g->np, g->stream));
        g->have_v = false;
    }
    CU(cudaStreamSynchronize(g->stream));
    return TDH_OK;
}

extern "C" int tdh_set_projectors(tdh_grid* g, int natoms, const int64_t* sph_off, const int32_t* sph_idx,
                                  const double* sph_disp, const int32_t* chan_off, const double* beta,
                                  const double* dcoef) {
    if (!g) return fail(TDH_EINVAL, "tdh_set_projectors: null handle");
    g->epoch += 1;
    if (natoms < 0) return fail(TDH_EINVAL, "tdh_set_projectors: natoms < 0");
    if (natoms == 0) {
        CU(cudaStreamSynchronize(g->stream));
        free_projectors(g);
        return TDH_OK;
    }
    // The new tables are validated and built first (host vectors, then device arrays of the staging handle `nw`); the
    // installed ones are replaced only when everything succeeded, so a rejected table leaves the handle as it was.
    if (natoms > 65535) return fail(TDH_EUNSUPPORTED, "tdh_set_projectors: more than 65535 atoms");
    if (!sph_off || !sph_idx || !chan_off || !beta || !dcoef)
        return fail(TDH_EINVAL, "tdh_set_projectors: null table with natoms > 0");
    if (g->have_k && !sph_disp) return fail(TDH_EINVAL, "tdh_set_projectors: sph_disp is required when k != 0");
    if (sph_off[0] != 0 || chan_off[0] != 0) return fail(TDH_EINVAL, "tdh_set_projectors: offsets must start at 0");
    for (int a = 0; a < natoms; ++a)
        if (sph_off[a + 1] < sph_off[a] || chan_off[a + 1] < chan_off[a])
            return fail(TDH_EINVAL, "tdh_set_projectors: offsets must be non-decreasing");
    const int64_t ptot = sph_off[natoms];
    const int ctot = chan_off[natoms];
    if (ctot == 0) {                       // atoms without any channel: V_nl = 0, the same as no projectors
        CU(cudaStreamSynchronize(g->stream));
        free_projectors(g);
        return TDH_OK;
    }
    if (ptot >= (int64_t)1 << 30) return fail(TDH_EUNSUPPORTED, "tdh_set_projectors: too many sphere points");

    // ---- validate, sort each sphere by flat grid index (coalesced gathers), re-index beta, build phases
    std::vector<int> stamp(g->np, -1);
    std::vector<int> sidx(ptot);
    std::vector<cd> sphase(g->have_k ? ptot : 0);
    std::vector<tdh::AtomDesc> atoms(natoms);
    std::vector<double> dscale(ctot);
    size_t btot = 0;
    int cmax = 0;
    for (int a = 0; a < natoms; ++a) {
        btot += (size_t)(chan_off[a + 1] - chan_off[a]) * (size_t)(sph_off[a + 1] - sph_off[a]);
        cmax = std::max(cmax, chan_off[a + 1] - chan_off[a]);
    }
    if (btot >= (size_t)1 << 31) return fail(TDH_EUNSUPPORTED, "tdh_set_projectors: projector table too large");
    if (cmax > 16) return fail(TDH_EUNSUPPORTED, "tdh_set_projectors: more than 16 channels on one atom");
    std::vector<double> sbeta(btot);
    std::vector<int> cover(g->np, 0);
    std::vector<int> order;
    size_t boff = 0;
    for (int a = 0; a < natoms; ++a) {
        const int64_t q0 = sph_off[a];
        const int pn = (int)(sph_off[a + 1] - q0);
        const int c0 = chan_off[a], nc = chan_off[a + 1] - c0;
        for (int q = 0; q < pn; ++q) {
            const int32_t p = sph_idx[q0 + q];
            if (p < 0 || (size_t)p >= g->np)
                return fail(TDH_EINDEX, "tdh_set_projectors: sph_idx[%lld] = %d out of range", (long long)(q0 + q), p);
            if (stamp[p] == a)
                return fail(TDH_EINDEX, "tdh_set_projectors: grid point %d listed twice for atom %d", p, a);
            stamp[p] = a;
            cover[p] += 1;
        }
        order.resize(pn);
        for (int q = 0; q < pn; ++q) order[q] = q;
        std::sort(order.begin(), order.end(), [&](int x, int y) { return sph_idx[q0 + x] < sph_idx[q0 + y]; });
        for (int j = 0; j < pn; ++j) {
            const int q = order[j];
            sidx[q0 + j] = sph_idx[q0 + q];
            if (g->have_k) {
                const double* d = sph_disp + 3 * (q0 + q);
                const double arg = g->kpt[0] * d[0] + g->kpt[1] * d[1] + g->kpt[2] * d[2];
                sphase[q0 + j] = make_double2(cos(arg), sin(arg));
            }
            for (int c = 0; c < nc; ++c) sbeta[boff + (size_t)c * pn + j] = beta[boff + (size_t)c * pn + q];
        }
        for (int c = 0; c < nc; ++c) dscale[c0 + c] = dcoef[c0 + c] * g->dv;
        atoms[a].q0 = (int)q0; atoms[a].np = pn; atoms[a].boff = (int)boff; atoms[a].chan0 = c0; atoms[a].nchan = nc;
        boff += (size_t)nc * pn;
    }
    // ---- z-runs of every sphere and their chunks (nl_kernels.cuh, nl_scatter_bulk_kernel): a run is a maximal sequence
    //      of consecutive flat indices of the sorted list, cut at SC_MAXPTS points; a chunk is up to SC_RC runs and
    //      SC_MAXPTS points, consecutive in the list
    std::vector<tdh::ScRun> sc_runs;
    std::vector<tdh::ScChunk> sc_chunks;
    for (int a = 0; a < natoms; ++a) {
        tdh::AtomDesc& at = atoms[a];
        at.sc0 = (int)sc_chunks.size();
        int j = 0;
        while (j < at.np) {
            int len = 1;
            while (j + len < at.np && len < tdh::SC_MAXPTS && sidx[at.q0 + j + len] == sidx[at.q0 + j] + len) ++len;
            if (sc_chunks.size() == (size_t)at.sc0 || sc_chunks.back().nr == tdh::SC_RC || sc_chunks.back().np + len > tdh::SC_MAXPTS)
                sc_chunks.push_back(tdh::ScChunk{(int)sc_runs.size(), 0, j, 0});
            tdh::ScChunk& ch = sc_chunks.back();
            sc_runs.push_back(tdh::ScRun{sidx[at.q0 + j], len, ch.np});
            ch.nr += 1;
            ch.np += len;
            j += len;
        }
        at.scn = (int)sc_chunks.size() - at.sc0;
    }
    // ---- colours for the separate back-projection kernel: greedy, an atom takes the lowest colour that no atom sharing
    //      a grid point with it has taken (per-point bit mask of the colours already present)
    std::vector<tdh::AtomDesc> atoms_col;
    std::vector<int> col_off;
    {
        std::vector<unsigned> pmask(g->np, 0u);
        std::vector<int> colour(natoms, 0);
        int ncol = 0;
        for (int a = 0; a < natoms; ++a) {
            unsigned used = 0u;
            for (int j = 0; j < atoms[a].np; ++j) used |= pmask[sidx[atoms[a].q0 + j]];
            int c = 0;
            while (c < 32 && (used >> c & 1u)) ++c;
            if (c == 32) return fail(TDH_EUNSUPPORTED, "tdh_set_projectors: more than 32 spheres overlap transitively at atom %d", a);
            colour[a] = c;
            ncol = std::max(ncol, c + 1);
            for (int j = 0; j < atoms[a].np; ++j) pmask[sidx[atoms[a].q0 + j]] |= 1u << c;
        }
        col_off.assign(ncol + 1, 0);
        for (int c = 0; c < ncol; ++c) {
            col_off[c] = (int)atoms_col.size();
            for (int a = 0; a < natoms; ++a)
                if (colour[a] == c) atoms_col.push_back(atoms[a]);
        }
        col_off[ncol] = (int)atoms_col.size();
    }
    // ---- back-projection records: one per (atom, sphere point), grouped by tile (x, r) and by layer.  The layer of a
    //      record is the number of earlier atoms covering the same grid point, so no two records of one (tile, layer)
    //      share a shared-memory cell and the scatter needs no atomics.  The cell address follows tile_kernels.cuh.
    if (ctot >= 65536) return fail(TDH_EUNSUPPORTED, "tdh_set_projectors: more than 65535 channels");
    const int ny = g->n[1], nz = g->n[2];
    const int S = g->tl.s, r1z = g->tl.r1z;
    int nlayers = 0;
    for (size_t p = 0; p < g->np; ++p) nlayers = std::max(nlayers, cover[p]);
    const int ntiles = g->n[0] * S;
    std::vector<int> nl_off((size_t)ntiles * (nlayers + 1) + 1, 0);
    std::vector<int> rec_slot(ptot);                       // (tile*(nlayers) + layer) of each (atom, point)
    std::vector<unsigned> rec_cell(ptot);
    {
        std::vector<int> fill(g->np, 0);
        std::vector<int> count((size_t)ntiles * nlayers, 0);
        for (int a = 0; a < natoms; ++a) {
            const tdh::AtomDesc& at = atoms[a];
            for (int j = 0; j < at.np; ++j) {
                const int p = sidx[at.q0 + j];
                const int x = p / (ny * nz), y = (p / nz) % ny, z = p % nz;
                const int r = y % S, m = y / S;
                const int line = m * r1z + (z >> 3);                 // natural order after the inverse transforms
                const int cell = 8 * line + ((z & 7) ^ (line & 7));  // tile_kernels.cuh, swz()
                const int layer = fill[p]++;
                const int slot = (x * S + r) * nlayers + layer;
                rec_slot[at.q0 + j] = slot;
                rec_cell[at.q0 + j] = (unsigned)cell | ((unsigned)at.chan0 << 16);
                count[slot] += 1;
            }
        }
        // offsets: tile t, layer l at nl_off[t*(nlayers+1) + l]; the end of the tile's last layer in [.. + nlayers]
        int run = 0;
        for (int t = 0; t < ntiles; ++t) {
            for (int l = 0; l < nlayers; ++l) { nl_off[(size_t)t * (nlayers + 1) + l] = run; run += count[(size_t)t * nlayers + l]; }
            nl_off[(size_t)t * (nlayers + 1) + nlayers] = run;
        }
    }
    const int cpad = tdh::nl_pad_cmax(cmax);               // channel count the record loop is compiled for
    std::vector<unsigned> rec_cc(ptot);
    std::vector<double> rec_beta((size_t)cpad * ptot, 0.0);
    std::vector<cd> rec_phase(g->have_k ? ptot : 0);
    {
        std::vector<int> cursor((size_t)ntiles * nlayers);
        for (int t = 0; t < ntiles; ++t)
            for (int l = 0; l < nlayers; ++l) cursor[(size_t)t * nlayers + l] = nl_off[(size_t)t * (nlayers + 1) + l];
        for (int a = 0; a < natoms; ++a) {
            const tdh::AtomDesc& at = atoms[a];
            for (int j = 0; j < at.np; ++j) {
                const int i = cursor[rec_slot[at.q0 + j]]++;
                rec_cc[i] = rec_cell[at.q0 + j];
                for (int c = 0; c < at.nchan; ++c) rec_beta[(size_t)c * ptot + i] = sbeta[at.boff + (size_t)c * at.np + j];
                if (g->have_k) rec_phase[i] = sphase[at.q0 + j];
            }
        }
    }

    auto up = [&](auto** dptr, const auto& vec) -> int {
        using T = typename std::remove_reference<decltype(vec)>::type::value_type;
        if (vec.empty()) { *dptr = nullptr; return TDH_OK; }
        CU(cudaMalloc(dptr, sizeof(T) * vec.size()));
        CU(cudaMemcpy(*dptr, vec.data(), sizeof(T) * vec.size(), cudaMemcpyHostToDevice));
        return TDH_OK;
    };
    int rc;
    tdh_grid stage{};                                      // only its projector fields are used
    tdh_grid* nw = &stage;
    if ((rc = up(&nw->d_sc_runs, sc_runs)) || (rc = up(&nw->d_sc_chunks, sc_chunks)) || (rc = up(&nw->d_atoms_col, atoms_col)) || (rc = up(&nw->d_atoms, atoms)) || (rc = up(&nw->d_sidx, sidx)) || (rc = up(&nw->d_sbeta, sbeta)) ||
        (rc = up(&nw->d_sphase, sphase)) || (rc = up(&nw->d_dscale, dscale)) || (rc = up(&nw->d_nl_off, nl_off)) ||
        (rc = up(&nw->d_nl_cc, rec_cc)) || (rc = up(&nw->d_nl_beta, rec_beta)) || (rc = up(&nw->d_nl_phase, rec_phase))) {
        free_projectors(nw);
        return rc;
    }
    // dpi: [chunk_cap][ctot] plus cpad zeroed entries (records of atoms with fewer than cpad channels read past their
    // own channels with a zero projector value)
    const size_t ndpi = (size_t)g->chunk_cap * ctot + cpad;
    cudaError_t e = cudaMalloc(&nw->d_dpi, sizeof(cd) * ndpi);
    if (e == cudaSuccess) e = cudaMemset(nw->d_dpi, 0, sizeof(cd) * ndpi);
    if (e != cudaSuccess) { free_projectors(nw); return fail(TDH_ENOMEM, "tdh_set_projectors: %s", cudaGetErrorString(e)); }
    {
        std::vector<double> dvs(ctot, g->dv);
        if ((rc = up(&nw->d_dvscale, dvs))) { free_projectors(nw); return rc; }
        e = cudaMalloc(&nw->d_dpig, sizeof(cd) * (size_t)g->chunk_cap * ctot);
        if (e == cudaSuccess && g->slab_world > 1) e = cudaMalloc(&nw->d_dpi_part, sizeof(cd) * (size_t)g->chunk_cap * ctot);
        if (e == cudaSuccess) e = cudaMalloc(&nw->d_force, sizeof(double) * (size_t)natoms * 3 * (1 + 64));
        if (e != cudaSuccess) { free_projectors(nw); return fail(TDH_ENOMEM, "tdh_set_projectors: %s", cudaGetErrorString(e)); }
    }
    // success: replace the installed tables
    if (cudaStreamSynchronize(g->stream) != cudaSuccess) { free_projectors(nw); return fail(TDH_ECUDA, "tdh_set_projectors: stream synchronisation failed"); }
    free_projectors(g);
    g->d_sc_runs = nw->d_sc_runs; g->d_sc_chunks = nw->d_sc_chunks;
    // Measured on B200 (profiles/r02_summary.md): runs of 12.8 points (Large) 4.10 ms by bulk reduce-add against 4.63 by
    // read-modify-write; runs of 8.6 points (TDDFT, forced onto the separate kernel) 0.347 against 0.334, Medium 0.141
    // against 0.129 -- one TMA operation per run and state pays from about ten points per run
    g->scatter_bulk = !sc_runs.empty() && (double)ptot / (double)sc_runs.size() >= 10.0;
    if (const char* e = getenv("TDH_SCATTER_BULK")) g->scatter_bulk = atoi(e) != 0;
    g->d_atoms_col = nw->d_atoms_col; g->d_atoms = nw->d_atoms; g->d_sidx = nw->d_sidx; g->d_sbeta = nw->d_sbeta;
    g->d_sphase = nw->d_sphase; g->d_dscale = nw->d_dscale; g->d_nl_off = nw->d_nl_off; g->d_nl_cc = nw->d_nl_cc;
    g->d_nl_beta = nw->d_nl_beta; g->d_nl_phase = nw->d_nl_phase; g->d_dpi = nw->d_dpi; g->d_dvscale = nw->d_dvscale;
    g->d_dpig = nw->d_dpig; g->d_force = nw->d_force; g->d_dpi_part = nw->d_dpi_part;
    if (g->slab_world > 1) {
        // the partial-projection buffer the peers were given has just been freed: no phase may run on the old addresses
        g->have_peers = false;
        for (int q = 0; q < tdh::SLAB_MAX_WORLD; ++q) g->peer_dpi[q] = nullptr;
    }
    g->natoms = natoms;
    g->nchan_tot = ctot;
    g->nl_layers = nlayers;
    g->nl_nrec = (int)ptot;
    g->nl_cmax = cpad;
    g->mt = cmax <= 8 ? 1 : 2;
    g->kt = (cmax + 3) / 4;
    g->col_off = col_off;
    // Measured on B200 (profiles/r01e_summary.md): the separate kernel wins on the split (half-plane) tiles of the large
    // grids, the records inside plane_inv win on whole-plane tiles.  TDH_NL_MODE=0/1 overrides (tests run both).
    g->nl_mode = g->tl.s == 2 ? 1 : 0;
    if (const char* e = getenv("TDH_NL_MODE")) g->nl_mode = atoi(e) != 0;
    if (g->generic) g->nl_mode = 1;                 // the record lists address tile cells: tuned grids only
    return TDH_OK;
}

// ------------------------------------------------------------------------------------------------------------
// launches
// ------------------------------------------------------------------------------------------------------------
static int prof_begin(tdh_grid* g, int k) {
    if (!g->profiling) return TDH_OK;
    if (g->prof_used == g->prof_pool.size()) {
        ProfRec r;
        CU(cudaEventCreate(&r.a));
        CU(cudaEventCreate(&r.b));
        r.k = k;
        g->prof_pool.push_back(r);
    }
    g->prof_pool[g->prof_used].k = k;
    CU(cudaEventRecord(g->prof_pool[g->prof_used].a, g->stream));
    return TDH_OK;
}
static int prof_end(tdh_grid* g) {
    if (!g->profiling) return TDH_OK;
    CU(cudaEventRecord(g->prof_pool[g->prof_used].b, g->stream));
    g->prof_used += 1;
    return TDH_OK;
}
static int prof_collect(tdh_grid* g) {
    if (!g->profiling) return TDH_OK;
    CU(cudaStreamSynchronize(g->stream));
    for (size_t i = 0; i < g->prof_used; ++i) {
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, g->prof_pool[i].a, g->prof_pool[i].b));
        g->ksec[g->prof_pool[i].k] += 1e-3 * ms;
    }
    g->prof_used = 0;
    return TDH_OK;
}
static void stats_reset(tdh_grid* g) {
    g->launch_count = 0;
    g->prof_used = 0;
    for (int i = 0; i < TDH_NKERNELS; ++i) g->ksec[i] = 0.0;
}

#define LAUNCH(kid, func, grid, block, smem, args)                                                 \
    do {                                                                                           \
        int rc_ = prof_begin(g, kid);                                                              \
        if (rc_) return rc_;                                                                       \
        CU(cudaLaunchKernel(func, grid, block, args, smem, g->stream));                            \
        g->launch_count += 1;                                                                      \
        rc_ = prof_end(g);                                                                         \
        if (rc_) return rc_;                                                                       \
    } while (0)

// CUtensorMap of a chunk of nst states starting at `base` as the tile kernels see it
static int tile_map(tdh_grid* g, const cd* base, int nst, CUtensorMap* m) {
    if (!tdh::encode_tile_map(m, base, (size_t)nst * g->n[0], g->n[1], g->n[2], g->tl.s, g->tl.ppc))
        return fail(TDH_ECUDA, "cuTensorMapEncodeTiled failed (tile map)");
    return TDH_OK;
}

// ---- general axis lengths (generic_fft.cuh): one batched 1-D transform per launch
// axis 0 = x, 1 = y, 2 = z of a block of nst states; dir = -1 / +1 plain transform (mode -1), or the x-pencil modes 0..4
static int launch_gaxis(tdh_grid* g, int kid, int nst, int axis, const cd* in, cd* out, int dir, int mode,
                        const double* tstate = nullptr) {
    tdh::GAxis ax = g->gax[axis];
    const size_t nx = g->n[0], ny = g->n[1], nz = g->n[2];
    if (axis == 2) { ax.stride = 1; ax.inner = 1; ax.outer = nz; ax.npencils = (size_t)nst * nx * ny; }
    else if (axis == 1) { ax.stride = nz; ax.inner = nz; ax.outer = ny * nz; ax.npencils = (size_t)nst * nx * nz; }
    else { ax.stride = ny * nz; ax.inner = ny * nz; ax.outer = nx * ny * nz; ax.npencils = (size_t)nst * ny * nz; }
    tdh::Kinetic kin;
    memset(&kin, 0, sizeof(kin));
    kin.g2x = g->d_g2[0]; kin.g2y_w = g->d_g2y_w; kin.g2z_w = g->d_g2z_w;
    if (mode == 3) { kin.g2x = g->d_p2x; kin.g2y_w = g->d_p2y_w; kin.g2z_w = g->d_p2z_w; }
    kin.tstate = tstate;
    kin.ecut = g->ecut;
    kin.scale = 1.0 / (double)g->np_total;
    kin.nz = g->n[2];
    kin.ny = g->n[1];
    const cd* tw = g->d_tw[axis];
    int nxi = g->n[0];
    const void* f = nullptr;
    switch (mode) {
        case -1: f = dir < 0 ? (const void*)&tdh::gfft_axis_kernel<-1, -1> : (const void*)&tdh::gfft_axis_kernel<+1, -1>; break;
        case 0: f = (const void*)&tdh::gfft_axis_kernel<-1, 0>; break;
        case 1: f = (const void*)&tdh::gfft_axis_kernel<-1, 1>; break;
        case 2: f = (const void*)&tdh::gfft_axis_kernel<-1, 2>; break;
        case 3: f = (const void*)&tdh::gfft_axis_kernel<-1, 3>; break;
        default: f = (const void*)&tdh::gfft_axis_kernel<-1, 4>; break;
    }
    void* args[] = {(void*)&in, (void*)&out, (void*)&ax, (void*)&tw, (void*)&kin, (void*)&nxi};
    const size_t tiles = (ax.npencils + ax.pt - 1) / ax.pt;
    // persistent grid: exactly the CTAs that are resident together (more would run as a second, partly empty wave)
    int occ = 0;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, f, tdh::GF_THREADS, tdh::gfft_smem(ax)));
    const unsigned grid = (unsigned)std::min<size_t>(tiles, (size_t)g->nsm * std::max(1, occ));
    LAUNCH(kid, f, dim3(grid), dim3(tdh::GF_THREADS), tdh::gfft_smem(ax), args);
    return TDH_OK;
}

static int launch_gzinv_epilogue(tdh_grid* g, int nst, const cd* in, cd* out, const tdh::Epilogue& ep) {
    tdh::GAxis ax = g->gax[2];
    ax.stride = 1; ax.inner = 1; ax.outer = g->n[2]; ax.npencils = (size_t)nst * g->n[0] * g->n[1];
    const cd* tw = g->d_tw[2];
    size_t npts = g->np;
    void* args[] = {(void*)&in, (void*)&out, (void*)&ax, (void*)&tw, (void*)&ep, (void*)&npts};
    const size_t tiles = (ax.npencils + ax.pt - 1) / ax.pt;
    int occ = 0;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void*)&tdh::gfft_zinv_epilogue_kernel, tdh::GF_THREADS,
                                                     tdh::gfft_smem(ax)));
    const unsigned grid = (unsigned)std::min<size_t>(tiles, (size_t)g->nsm * std::max(1, occ));
    LAUNCH(K_PLANE_INV, (const void*)&tdh::gfft_zinv_epilogue_kernel, dim3(grid), dim3(tdh::GF_THREADS), tdh::gfft_smem(ax), args);
    return TDH_OK;
}

// to_peers (slab handles): every spectrum row is stored into the Fourier-space slab of the rank that owns it
static int launch_plane_fwd(tdh_grid* g, int nst, const cd* in, cd* out, bool to_peers = false) {
    if (g->generic) {
        int rc = launch_gaxis(g, K_PLANE_FWD, nst, 2, in, out, -1, -1);
        return rc ? rc : launch_gaxis(g, K_PLANE_FWD, nst, 1, out, out, -1, -1);
    }
    CUtensorMap map;
    int rc = tile_map(g, in, nst, &map);
    if (rc) return rc;
    const cd* twy = g->d_tw[1];
    const cd* twz = g->d_tw[2];
    int ntiles = (int)((size_t)nst * g->n[0] * g->tl.s / g->tl.ppc);
    tdh::SlabDst sd;
    memset(&sd, 0, sizeof(sd));
    if (to_peers) {
        for (int q = 0; q < g->slab_world; ++q) sd.fs[q] = g->peer_fs[q];
        sd.ny_local = g->ny_local; sd.nx_local = g->n[0]; sd.nx_total = g->nx_fs; sd.x0 = g->slab_rank * g->n[0];
    }
    void* args[] = {(void*)&map, (void*)&out, (void*)&ntiles, (void*)&twy, (void*)&twz, (void*)&sd};
    const unsigned grid = (unsigned)std::min(ntiles, to_peers ? g->ctas_fwd_slab : g->ctas_fwd);
    LAUNCH(K_PLANE_FWD, to_peers ? g->tl.fwd_slab : g->tl.fwd, dim3(grid), dim3(g->tl.threads), g->tl.smem_fwd, args);
    return TDH_OK;
}

// On a slab handle `in` is this rank's Fourier-space slab [nst][NX][ny_local][NZ]; with to_peers (modes 0 and 2) the
// values of plane x are stored into the real-space work buffer of the rank that owns x.
static int launch_xpencil(tdh_grid* g, int nst, const cd* in, cd* out, int mode, const double* tstate = nullptr,
                          bool to_peers = false) {
    if (g->generic) return launch_gaxis(g, K_XPENCIL, nst, 0, in, out, -1, mode, tstate);
    const bool slab = g->slab_world > 1;
    const int ny = slab ? g->ny_local : g->n[1];                     // rows of the block this launch sees
    const int y0 = slab ? g->slab_rank * g->ny_local : 0;
    CUtensorMap map;
    if (!tdh::encode_line_map(&map, in, (size_t)nst * g->nx_fs, g->nx_fs, ny, g->n[2]))
        return fail(TDH_ECUDA, "cuTensorMapEncodeTiled failed (line map)");
    tdh::Kinetic kin;
    kin.g2x = g->d_g2[0]; kin.g2y_w = g->d_g2y_w + y0; kin.g2z_w = g->d_g2z_w; kin.twy_w = g->d_twy_w + y0 / 2;
    if (mode == 3) { kin.g2x = g->d_p2x; kin.g2y_w = g->d_p2y_w + y0; kin.g2z_w = g->d_p2z_w; }     // Poisson: pure |G|^2
    kin.tstate = tstate;
    kin.ecut = g->ecut;
    kin.scale = 1.0 / (double)g->np_total;
    kin.nz = g->n[2];
    kin.ny = ny;
    int ntiles = nst * (ny / 2) * (g->n[2] / 16);
    const cd* twx = g->d_tw[0];
    tdh::SlabSrc ss;
    memset(&ss, 0, sizeof(ss));
    const void* f = mode == 0 ? g->xl.fused : (mode == 1 ? g->xl.fwd : (mode == 2 ? g->xl.inv : (mode == 3 ? g->xl.poisson : g->xl.teter)));
    int ctas = g->ctas_x[mode];
    if (to_peers) {
        if (mode != 0 && mode != 2) return fail(TDH_EINVAL, "launch_xpencil: no slab stores for mode %d", mode);
        for (int q = 0; q < g->slab_world; ++q) ss.rs[q] = g->peer_rs[q];
        ss.nx_local = g->n[0]; ss.ny_total = g->n[1]; ss.y0 = y0;
        f = mode == 0 ? g->xl.fused_slab : g->xl.inv_slab;
        ctas = g->ctas_x_slab[mode == 0 ? 0 : 1];
    }
    void* args[] = {(void*)&map, (void*)&out, (void*)&ntiles, (void*)&twx, (void*)&kin, (void*)&ss};
    const unsigned grid = (unsigned)std::min(ntiles, ctas);
    LAUNCH(K_XPENCIL, f, dim3(grid), dim3(g->xl.threads), g->xl.smem, args);
    return TDH_OK;
}

// in: work block (spectrum), phi: input block of this application (read only when the epilogue has V or projectors)
static int launch_plane_inv(tdh_grid* g, int nst, const cd* in, const cd* phi, cd* out, const tdh::Epilogue& ep) {
    if (g->generic) {
        // `in` is always one of the handle's scratch blocks: the y transform runs in place on it
        cd* w = const_cast<cd*>(in);
        int rc = launch_gaxis(g, K_PLANE_INV, nst, 1, w, w, +1, -1);
        if (rc) return rc;
        tdh::Epilogue epl = ep;
        epl.phi = phi;
        return launch_gzinv_epilogue(g, nst, w, out, epl);
    }
    CUtensorMap map_spec, map_phi;
    int rc = tile_map(g, in, nst, &map_spec);
    if (rc) return rc;
    if ((rc = tile_map(g, phi ? phi : in, nst, &map_phi))) return rc;
    CUtensorMap map_yv;
    if ((rc = tile_map(g, ep.yv ? ep.yv : in, nst, &map_yv))) return rc;
    const cd* twy = g->d_tw[1];
    const cd* twz = g->d_tw[2];
    int ntiles = (int)((size_t)nst * g->n[0] * g->tl.s / g->tl.ppc);
    tdh::Epilogue epl = ep;
    epl.phi = phi;
    void* args[] = {(void*)&map_spec, (void*)&map_phi, (void*)&map_yv, (void*)&out, (void*)&ntiles, (void*)&twy, (void*)&twz, (void*)&epl};
    const int cmi = tdh::nl_cm_index(epl.nl_off != nullptr ? epl.cmax : 0);
    const unsigned grid = (unsigned)std::min(ntiles, g->ctas_inv[cmi]);
    LAUNCH(K_PLANE_INV, g->tl.inv[cmi], dim3(grid), dim3(g->tl.threads), g->tl.smem_inv, args);
    return TDH_OK;
}

// natural (ky, kz) order <-> work layout, for tdh_fft3d only.  dir 0: out[plane][ky][kz] = in[plane][rowmap[ky]][colmap[kz]];
// dir 1: the inverse permutation.
__global__ void reorder_kernel(const cd* __restrict__ in, cd* __restrict__ out, size_t nplanes, int ny, int nz,
                               const int* __restrict__ rowmap, const int* __restrict__ colmap, int dir) {
    const size_t total = nplanes * ny * nz;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int kz = (int)(i % nz), ky = (int)((i / nz) % ny);
        const size_t plane = i / ((size_t)ny * nz);
        const size_t j = (plane * ny + rowmap[ky]) * nz + colmap[kz];
        if (dir == 0) out[i] = in[j]; else out[j] = in[i];
    }
}

static int launch_reorder(tdh_grid* g, int nst, const cd* in, cd* out, int dir) {
    const size_t nplanes = (size_t)nst * g->n[0];
    reorder_kernel<<<1184, 256, 0, g->stream>>>(in, out, nplanes, g->n[1], g->n[2], g->d_rowmap, g->d_colmap, dir);
    CU(cudaGetLastError());
    g->launch_count += 1;
    return TDH_OK;
}

static int launch_nl_project(tdh_grid* g, int nst, const cd* in, const double* dscale_in = nullptr, cd* dpi_out = nullptr) {
    size_t npts = g->np;
    const tdh::AtomDesc* atoms = g->d_atoms;
    const int* sidx = g->d_sidx;
    const double* sbeta = g->d_sbeta;
    const cd* sphase = g->d_sphase;
    const double* dscale = dscale_in ? dscale_in : g->d_dscale;
    cd* dpi = dpi_out ? dpi_out : (g->slab_world > 1 ? g->d_dpi_part : g->d_dpi);
    int nct = g->nchan_tot;
    void* args[] = {(void*)&in, (void*)&npts, (void*)&nst, (void*)&atoms, (void*)&sidx, (void*)&sbeta,
                    (void*)&sphase, (void*)&dscale, (void*)&dpi, (void*)&nct};
    const void* f = g->mt == 1 ? reinterpret_cast<const void*>(&tdh::nl_project_kernel<1>)
                               : reinterpret_cast<const void*>(&tdh::nl_project_kernel<2>);
    dim3 grid(g->natoms, (nst + tdh::NLP_STATES - 1) / tdh::NLP_STATES);
    LAUNCH(K_NLPROJ, f, grid, dim3(32 * tdh::NLP_WARPS), 0, args);
    return TDH_OK;
}

// out += alpha * V_nl phi from the coefficients nl_project left in d_dpi: one launch per colour
static int launch_nl_scatter(tdh_grid* g, int nst, cd* out, cd alpha) {
    size_t npts = g->np;
    const int* sidx = g->d_sidx;
    const double* sbeta = g->d_sbeta;
    const cd* sphase = g->d_sphase;
    const cd* dpi = g->d_dpi;
    int nct = g->nchan_tot;
    const void* fs[4] = {reinterpret_cast<const void*>(&tdh::nl_scatter_kernel<1>), reinterpret_cast<const void*>(&tdh::nl_scatter_kernel<2>),
                         reinterpret_cast<const void*>(&tdh::nl_scatter_kernel<3>), reinterpret_cast<const void*>(&tdh::nl_scatter_kernel<4>)};
    if (g->kt < 1) return TDH_OK;                          // no channel anywhere: nothing to add
    if (g->scatter_bulk) {
        // the read-modify-write done by the L2: one bulk reduce-add per (z-run, state) (nl_kernels.cuh)
        const void* fb[4] = {reinterpret_cast<const void*>(&tdh::nl_scatter_bulk_kernel<1>), reinterpret_cast<const void*>(&tdh::nl_scatter_bulk_kernel<2>),
                             reinterpret_cast<const void*>(&tdh::nl_scatter_bulk_kernel<3>), reinterpret_cast<const void*>(&tdh::nl_scatter_bulk_kernel<4>)};
        const tdh::ScRun* runs = g->d_sc_runs;
        const tdh::ScChunk* chunks = g->d_sc_chunks;
        for (size_t c = 0; c + 1 < g->col_off.size(); ++c) {
            const tdh::AtomDesc* atoms = g->d_atoms_col + g->col_off[c];
            void* args[] = {(void*)&out, (void*)&npts, (void*)&nst, (void*)&atoms, (void*)&runs, (void*)&chunks, (void*)&sbeta,
                            (void*)&sphase, (void*)&dpi, (void*)&nct, (void*)&alpha};
            dim3 grid(g->col_off[c + 1] - g->col_off[c], (nst + tdh::NLP_STATES - 1) / tdh::NLP_STATES);
            LAUNCH(K_NLSCATTER, fb[g->kt - 1], grid, dim3(32 * tdh::NLS_WARPS), tdh::SC_SMEM, args);
        }
        return TDH_OK;
    }
    for (size_t c = 0; c + 1 < g->col_off.size(); ++c) {
        const tdh::AtomDesc* atoms = g->d_atoms_col + g->col_off[c];
        void* args[] = {(void*)&out, (void*)&npts, (void*)&nst, (void*)&atoms, (void*)&sidx, (void*)&sbeta,
                        (void*)&sphase, (void*)&dpi, (void*)&nct, (void*)&alpha};
        dim3 grid(g->col_off[c + 1] - g->col_off[c], (nst + tdh::NLP_STATES - 1) / tdh::NLP_STATES);
        LAUNCH(K_NLSCATTER, fs[g->kt - 1], grid, dim3(32 * tdh::NLS_WARPS), 0, args);
    }
    return TDH_OK;
}

static int finish_chunk(tdh_grid* g, int nst, const cd* in, cd* out, cd alpha, const cd* yv);
static int launch_small(tdh_grid* g, int nst, const cd* in, cd* out, cd alpha, const cd* yv);

// out = alpha * H in + yv   for one chunk (nst <= chunk_cap); in/out/yv point at the chunk's first state
static int apply_chunk(tdh_grid* g, int nst, const cd* in, cd* out, cd alpha, const cd* yv, bool kinetic_only = false) {
    int rc;
    if (kinetic_only) {                                   // out = alpha * T in + yv
        if ((rc = launch_plane_fwd(g, nst, in, g->d_work))) return rc;
        if ((rc = launch_xpencil(g, nst, g->d_work, g->d_work, 0))) return rc;
        tdh::Epilogue ek;
        memset(&ek, 0, sizeof(ek));
        ek.yv = yv;
        ek.alpha = alpha;
        ek.nx = g->n[0];
        return launch_plane_inv(g, nst, g->d_work, nullptr, out, ek);
    }
    if (g->small_cs > 0 && g->nchan_tot <= tdh::SMALL_MAX_CHAN) return launch_small(g, nst, in, out, alpha, yv);
    if (g->natoms > 0 && (rc = launch_nl_project(g, nst, in))) return rc;
    if ((rc = launch_plane_fwd(g, nst, in, g->d_work))) return rc;
    if ((rc = launch_xpencil(g, nst, g->d_work, g->d_work, 0))) return rc;
    return finish_chunk(g, nst, in, out, alpha, yv);
}

// the whole application in one launch: a CTA (16^3) or a cluster of four CTAs (32^3) per state (small_kernels.cuh)
static int launch_small(tdh_grid* g, int nst, const cd* in, cd* out, cd alpha, const cd* yv) {
    tdh::Kinetic kin;
    memset(&kin, 0, sizeof(kin));
    kin.g2x = g->d_g2[0]; kin.g2y_w = g->d_g2y_w; kin.g2z_w = g->d_g2z_w;
    kin.ecut = g->ecut;
    kin.scale = 1.0 / (double)g->np_total;
    kin.nz = g->n[2];
    kin.ny = g->n[1];
    tdh::Epilogue ep;
    memset(&ep, 0, sizeof(ep));
    ep.v = g->have_v ? g->d_v : nullptr;
    ep.phi = in;
    ep.yv = yv;
    ep.alpha = alpha;
    ep.nx = g->n[0];
    tdh::SmallProj pj;
    memset(&pj, 0, sizeof(pj));
    if (g->natoms > 0) {
        ep.nl_off = g->d_nl_off; ep.nl_layers = g->nl_layers; ep.nl_cc = g->d_nl_cc; ep.nl_beta = g->d_nl_beta;
        ep.nl_phase = g->d_nl_phase; ep.nrec = g->nl_nrec; ep.cmax = g->nl_cmax; ep.nchan_tot = g->nchan_tot;
        pj.atoms = g->d_atoms; pj.sidx = g->d_sidx; pj.sbeta = g->d_sbeta; pj.sphase = g->d_sphase; pj.dscale = g->d_dscale;
        pj.natoms = g->natoms; pj.nchan_tot = g->nchan_tot;
    }
    const cd* twx = g->d_tw[0];
    const cd* twy = g->d_tw[1];
    const cd* twz = g->d_tw[2];
    void* args[] = {(void*)&in, (void*)&out, (void*)&twx, (void*)&twy, (void*)&twz, (void*)&kin, (void*)&ep, (void*)&pj};
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    // 16^3 with few states: a cluster of four CTAs per state (the machine is mostly idle with one CTA per state, and a
    // pass over a quarter of the state is a quarter of the latency); with many states one CTA per state (no DSMEM stage)
    int cs = g->small_cs, cells = g->small_cells;
    const void* fn = g->small_fn;
    if (g->small_cs == 1 && g->small16_cluster && nst * 4 <= g->nsm) {
        cs = 4; cells = tdh::SmallCfg<16, 4>::CELLS; fn = (const void*)&tdh::small_h_kernel<16, 4>;
    }
    cfg.gridDim = dim3((unsigned)(nst * cs));
    cfg.blockDim = dim3(g->small_cs == 1 ? tdh::SmallCfg<16, 1>::T : tdh::SmallCfg<32, 4>::T);
    cfg.dynamicSmemBytes = tdh::small_smem(cells, g->natoms, g->nchan_tot);
    cfg.stream = g->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)cs;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    int rc_ = prof_begin(g, K_SMALL_H);
    if (rc_) return rc_;
    CU(cudaLaunchKernelExC(&cfg, fn, args));
    g->launch_count += 1;
    return prof_end(g);
}

// last part of one application: inverse (y,z) transform of the work block with the fused epilogue (+ back-projection)
static int finish_chunk(tdh_grid* g, int nst, const cd* in, cd* out, cd alpha, const cd* yv) {
    int rc;
    tdh::Epilogue ep;
    memset(&ep, 0, sizeof(ep));
    const bool fused_nl = g->natoms > 0 && g->nl_mode == 0;
    ep.v = (g->have_v || fused_nl) ? g->d_v : nullptr;        // zero-filled until set; required with the fused records
    ep.yv = yv;
    ep.alpha = alpha;
    ep.nx = g->n[0];
    if (fused_nl) {
        ep.nl_off = g->d_nl_off;
        ep.nl_layers = g->nl_layers;
        ep.nl_cc = g->d_nl_cc;
        ep.nl_beta = g->d_nl_beta;
        ep.nl_phase = g->d_nl_phase;
        ep.dpi = g->d_dpi;
        ep.nrec = g->nl_nrec;
        ep.cmax = g->nl_cmax;
        ep.nchan_tot = g->nchan_tot;
    }
    if ((rc = launch_plane_inv(g, nst, g->d_work, in, out, ep))) return rc;
    if (g->natoms > 0 && !fused_nl) return launch_nl_scatter(g, nst, out, alpha);
    return TDH_OK;
}

static int apply_block(tdh_grid* g, int nst, const cd* psi, cd* hpsi) {
    for (int s0 = 0; s0 < nst; s0 += g->chunk) {
        const int c = std::min(g->chunk, nst - s0);
        int rc = apply_chunk(g, c, psi + (size_t)s0 * g->np, hpsi + (size_t)s0 * g->np, make_double2(1.0, 0.0), nullptr);
        if (rc) return rc;
    }
    return TDH_OK;
}

// all steps of one chunk, Horner form of Eq. 8
static int propagate_chunk(tdh_grid* g, int nst, cd* psi, double dt, int nsteps) {
    cd* pa = g->d_phi[0];
    cd* pb = g->d_phi[1];
    for (int step = 0; step < nsteps; ++step) {
        int rc;
        if ((rc = apply_chunk(g, nst, psi, pa, make_double2(0.0, -dt / 4.0), psi))) return rc;
        if ((rc = apply_chunk(g, nst, pa, pb, make_double2(0.0, -dt / 3.0), psi))) return rc;
        if ((rc = apply_chunk(g, nst, pb, pa, make_double2(0.0, -dt / 2.0), psi))) return rc;
        if ((rc = apply_chunk(g, nst, pa, psi, make_double2(0.0, -dt), psi))) return rc;
    }
    return TDH_OK;
}

// half = psi + sum_k a_k phi_k (written over psi), full = psi + sum_k b_k phi_k (written over phi_1), k = 1..4, elementwise
__global__ void taylor_pair_combine_kernel(cd* __restrict__ psi, cd* __restrict__ f1, const cd* __restrict__ p2,
                                           const cd* __restrict__ p3, const cd* __restrict__ p4, size_t n, cd a1, cd a2,
                                           cd a3, cd a4, cd b1, cd b2, cd b3, cd b4) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const cd x = __ldcs(psi + i), y1 = __ldcs(f1 + i), y2 = __ldcs(p2 + i), y3 = __ldcs(p3 + i), y4 = __ldcs(p4 + i);
        cd h = tdh::cfma(a1, y1, x), f = tdh::cfma(b1, y1, x);
        h = tdh::cfma(a2, y2, h); f = tdh::cfma(b2, y2, f);
        h = tdh::cfma(a3, y3, h); f = tdh::cfma(b3, y3, f);
        h = tdh::cfma(a4, y4, h); f = tdh::cfma(b4, y4, f);
        __stcs(psi + i, h);
        __stcs(f1 + i, f);
    }
}

// phi_k = H phi_{k-1} once, both Taylor sums from the same four vectors.  Runs in half chunks so that
// phi_2, phi_3 (halves of d_phi[0]) and phi_4 (d_phi[1]) fit the handle's workspace; phi_1 lives in the caller's `full`.
static int taylor_pair_block(tdh_grid* g, int nst, cd* psi, cd* full, double dt) {
    const int hc = std::max(1, g->chunk / 2);
    const cd one = make_double2(1.0, 0.0);
    // (-i dt)^k / k!  and  (-i dt/2)^k / k!
    const double d = dt, e = 0.5 * dt;
    const cd b1 = make_double2(0.0, -d), b2 = make_double2(-d * d / 2.0, 0.0), b3 = make_double2(0.0, d * d * d / 6.0),
             b4 = make_double2(d * d * d * d / 24.0, 0.0);
    const cd a1 = make_double2(0.0, -e), a2 = make_double2(-e * e / 2.0, 0.0), a3 = make_double2(0.0, e * e * e / 6.0),
             a4 = make_double2(e * e * e * e / 24.0, 0.0);
    for (int s0 = 0; s0 < nst; s0 += hc) {
        const int c = std::min(hc, nst - s0);
        cd* x = psi + (size_t)s0 * g->np;
        cd* f1 = full + (size_t)s0 * g->np;
        cd* p2 = g->d_phi[0];
        cd* p3 = g->d_phi[0] + (size_t)hc * g->np;
        cd* p4 = g->d_phi[1];
        int rc;
        if ((rc = apply_chunk(g, c, x, f1, one, nullptr))) return rc;
        if ((rc = apply_chunk(g, c, f1, p2, one, nullptr))) return rc;
        if ((rc = apply_chunk(g, c, p2, p3, one, nullptr))) return rc;
        if ((rc = apply_chunk(g, c, p3, p4, one, nullptr))) return rc;
        const size_t n = (size_t)c * g->np;
        taylor_pair_combine_kernel<<<148 * 8, 256, 0, g->stream>>>(x, f1, p2, p3, p4, n, a1, a2, a3, a4, b1, b2, b3, b4);
        CU(cudaGetLastError());
        g->launch_count += 1;
    }
    return TDH_OK;
}

static int propagate_block(tdh_grid* g, int nst, cd* psi, double dt, int nsteps) {
    for (int s0 = 0; s0 < nst; s0 += g->chunk) {
        const int c = std::min(g->chunk, nst - s0);
        int rc = propagate_chunk(g, c, psi + (size_t)s0 * g->np, dt, nsteps);
        if (rc) return rc;
    }
    return TDH_OK;
}

// entry points that transform along x need the whole grid on one device: refused on the handles of a slab decomposition
#define NOT_SLAB(name)                                                                                        \
    do {                                                                                                      \
        if (g->slab_world > 1) return fail(TDH_EINVAL, name ": not available on a slab handle (tdh_slab_*)"); \
    } while (0)

static bool overlaps(const void* a, const void* b, size_t bytes) {
    const char* x = (const char*)a;
    const char* y = (const char*)b;
    return x < y + bytes && y < x + bytes;
}

extern "C" int tdh_apply_hamiltonian(tdh_grid* g, int nst, const tdh_c128* psi_dev, tdh_c128* hpsi_dev) {
    if (!g || !psi_dev || !hpsi_dev) return fail(TDH_EINVAL, "tdh_apply_hamiltonian: null argument");
    NOT_SLAB("tdh_apply_hamiltonian");
    if (nst < 1 || nst > g->max_states) return fail(TDH_EINVAL, "tdh_apply_hamiltonian: nst = %d outside [1, %d]", nst, g->max_states);
    if (overlaps(psi_dev, hpsi_dev, (size_t)nst * g->np * sizeof(cd)))
        return fail(TDH_EINVAL, "tdh_apply_hamiltonian: psi and hpsi overlap");
    stats_reset(g);
    int rc = apply_block(g, nst, (const cd*)psi_dev, (cd*)hpsi_dev);
    if (rc) return rc;
    return prof_collect(g);
}

extern "C" int tdh_propagate(tdh_grid* g, int nst, tdh_c128* psi_dev, double dt, int nsteps, int order) {
    if (!g || !psi_dev) return fail(TDH_EINVAL, "tdh_propagate: null argument");
    NOT_SLAB("tdh_propagate");
    if (nst < 1 || nst > g->max_states) return fail(TDH_EINVAL, "tdh_propagate: nst = %d outside [1, %d]", nst, g->max_states);
    if (order != 4) return fail(TDH_EINVAL, "tdh_propagate: order must be 4");
    if (nsteps < 0 || !std::isfinite(dt)) return fail(TDH_EINVAL, "tdh_propagate: bad dt / nsteps");
    stats_reset(g);
    // Small blocks are bound by launch latency (Tiny: one 9 us kernel per application): replay the call as one CUDA graph.
    // Captured on an internal stream (the caller's may be the legacy default stream, which cannot capture), launched on
    // the caller's.  Kernel arguments, tensor maps included, are frozen in the graph, hence the key below.
    const size_t block_bytes = (size_t)nst * g->np * sizeof(cd);
    const long nodes = (long)nsteps * 4 * 6 * ((nst + g->chunk - 1) / g->chunk);
    if (g->use_graph && !g->profiling && nsteps > 0 && block_bytes <= ((size_t)128 << 20) && nodes <= 8192) {
        tdh_grid::PropGraph* pg = nullptr;
        for (auto& e : g->pg)
            if (e.exec && e.psi == (const void*)psi_dev && e.nst == nst && e.nsteps == nsteps && e.dt == dt && e.epoch == g->epoch) pg = &e;
        if (!pg) {
            tdh_grid::PropGraph& e = g->pg[g->pg_next];
            g->pg_next = (g->pg_next + 1) % 4;
            if (e.exec) { CU(cudaStreamSynchronize(g->stream)); cudaGraphExecDestroy(e.exec); e.exec = nullptr; }   // not while it may run
            if (!g->s_cap) CU(cudaStreamCreateWithFlags(&g->s_cap, cudaStreamNonBlocking));
            cudaStream_t user = g->stream;
            g->stream = g->s_cap;
            cudaGraph_t graph = nullptr;
            cudaError_t ce = cudaStreamBeginCapture(g->s_cap, cudaStreamCaptureModeThreadLocal);
            int rc = ce == cudaSuccess ? propagate_block(g, nst, (cd*)psi_dev, dt, nsteps) : TDH_ECUDA;
            if (ce == cudaSuccess) ce = cudaStreamEndCapture(g->s_cap, &graph);
            g->stream = user;
            if (rc == TDH_OK && ce == cudaSuccess && graph) ce = cudaGraphInstantiate(&e.exec, graph, 0);
            if (graph) cudaGraphDestroy(graph);
            if (rc != TDH_OK || ce != cudaSuccess || !e.exec) {
                (void)cudaGetLastError();                 // capture is an optimisation: fall back to plain launches
                e.exec = nullptr;
                g->use_graph = false;
            } else {
                e.psi = psi_dev; e.nst = nst; e.nsteps = nsteps; e.dt = dt; e.epoch = g->epoch;
                e.launches = g->launch_count;
                pg = &e;
            }
        }
        if (pg) {
            CU(cudaGraphLaunch(pg->exec, g->stream));
            g->launch_count = pg->launches;
            return TDH_OK;
        }
        stats_reset(g);
    }
    int rc = propagate_block(g, nst, (cd*)psi_dev, dt, nsteps);
    if (rc) return rc;
    return prof_collect(g);
}

extern "C" int tdh_taylor_pair(tdh_grid* g, int nst, tdh_c128* psi_dev, tdh_c128* full_dev, double dt, int order) {
    if (!g || !psi_dev || !full_dev) return fail(TDH_EINVAL, "tdh_taylor_pair: null argument");
    NOT_SLAB("tdh_taylor_pair");
    if (nst < 1 || nst > g->max_states) return fail(TDH_EINVAL, "tdh_taylor_pair: nst = %d outside [1, %d]", nst, g->max_states);
    if (order != 4) return fail(TDH_EINVAL, "tdh_taylor_pair: order must be 4");
    if (!std::isfinite(dt)) return fail(TDH_EINVAL, "tdh_taylor_pair: bad dt");
    if (overlaps(psi_dev, full_dev, (size_t)nst * g->np * sizeof(cd)))
        return fail(TDH_EINVAL, "tdh_taylor_pair: psi and full overlap");
    stats_reset(g);
    int rc = taylor_pair_block(g, nst, (cd*)psi_dev, (cd*)full_dev, dt);
    if (rc) return rc;
    return prof_collect(g);
}

extern "C" int tdh_etrs_step(tdh_grid* g, int nst, tdh_c128* psi_dev, tdh_c128* approx_dev, double dt,
                             const double* v_next_dev) {
    if (!g || !psi_dev || !approx_dev) return fail(TDH_EINVAL, "tdh_etrs_step: null argument");
    NOT_SLAB("tdh_etrs_step");
    if (nst < 1 || nst > g->max_states) return fail(TDH_EINVAL, "tdh_etrs_step: nst = %d outside [1, %d]", nst, g->max_states);
    if (!std::isfinite(dt)) return fail(TDH_EINVAL, "tdh_etrs_step: bad dt");
    if (overlaps(psi_dev, approx_dev, (size_t)nst * g->np * sizeof(cd)))
        return fail(TDH_EINVAL, "tdh_etrs_step: psi and approx overlap");
    stats_reset(g);
    int rc = taylor_pair_block(g, nst, (cd*)psi_dev, (cd*)approx_dev, dt);          // Eq. 7 and the first factor of Eq. 6
    if (rc) return rc;
    // H(t+dt): stream-ordered switch of the potential
    g->epoch += 1;
    if (v_next_dev) {
        CU(cudaMemcpyAsync(g->d_v, v_next_dev, sizeof(double) * g->np, cudaMemcpyDeviceToDevice, g->stream));
        g->have_v = true;
    } else {
        CU(cudaMemsetAsync(g->d_v, 0, sizeof(double) * g->np, g->stream));
        g->have_v = false;
    }
    const int launches = g->launch_count;
    if ((rc = propagate_block(g, nst, (cd*)psi_dev, 0.5 * dt, 1))) return rc;      // the second factor of Eq. 6
    (void)launches;
    return prof_collect(g);
}

// ------------------------------------------------------------------------------------------------------------
// NEXT-2: density (Eq. 1) and periodic Hartree potential
// ------------------------------------------------------------------------------------------------------------
// n[p] (+)= sum_s occ[s] |psi_s[p]|^2.  One thread per grid point (consecutive threads read consecutive 16-byte values of
// one state), states summed in order: deterministic, the order of the oracle.  Eight loads in flight per thread.
__global__ void density_kernel(const cd* __restrict__ psi, size_t npts, int nst, const double* __restrict__ occ,
                               double* __restrict__ dens, int accumulate) {
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npts) return;
    double acc = accumulate ? dens[p] : 0.0;
    int s = 0;
    for (; s + 8 <= nst; s += 8) {
        cd v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) v[u] = __ldcs(psi + (size_t)(s + u) * npts + p);
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const double a = __dadd_rn(__dmul_rn(v[u].x, v[u].x), __dmul_rn(v[u].y, v[u].y));
            acc = __dadd_rn(acc, __dmul_rn(occ ? occ[s + u] : 1.0, a));
        }
    }
    for (; s < nst; ++s) {
        const cd v = __ldcs(psi + (size_t)s * npts + p);
        const double a = __dadd_rn(__dmul_rn(v.x, v.x), __dmul_rn(v.y, v.y));
        acc = __dadd_rn(acc, __dmul_rn(occ ? occ[s] : 1.0, a));
    }
    dens[p] = acc;
}

__global__ void real_to_complex_kernel(const double* __restrict__ in, cd* __restrict__ out, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        out[i] = make_double2(in[i], 0.0);
}
__global__ void complex_to_real_kernel(const cd* __restrict__ in, double* __restrict__ out, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        out[i] = in[i].x;
}

extern "C" int tdh_density(tdh_grid* g, int nst, const tdh_c128* psi_dev, const double* occ_host, double* n_dev,
                           int accumulate) {
    if (!g || !psi_dev || !n_dev) return fail(TDH_EINVAL, "tdh_density: null argument");
    if (nst < 1 || nst > g->max_states) return fail(TDH_EINVAL, "tdh_density: nst = %d outside [1, %d]", nst, g->max_states);
    stats_reset(g);
    const double* occ = nullptr;
    if (occ_host) {
        // stream-ordered after the kernels that may still read the previous occupations
        CU(cudaMemcpyAsync(g->d_occ, occ_host, sizeof(double) * nst, cudaMemcpyHostToDevice, g->stream));
        CU(cudaStreamSynchronize(g->stream));             // occ_host may be pageable and reused by the caller
        occ = g->d_occ;
    }
    const unsigned blocks = (unsigned)((g->np + 255) / 256);
    density_kernel<<<blocks, 256, 0, g->stream>>>((const cd*)psi_dev, g->np, nst, occ, n_dev, accumulate);
    CU(cudaGetLastError());
    g->launch_count += 1;
    return TDH_OK;
}

// v_H: real -> complex, forward (z,y), x-pencil pass with the Poisson factor, inverse (y,z), real part.  One state's
// worth of work through the same three FFT kernels as H; uses the work buffer and the first Horner buffer.
extern "C" int tdh_hartree(tdh_grid* g, const double* n_dev, double* vh_dev) {
    if (!g || !n_dev || !vh_dev) return fail(TDH_EINVAL, "tdh_hartree: null argument");
    NOT_SLAB("tdh_hartree");
    stats_reset(g);
    cd* a = g->d_phi[0];
    real_to_complex_kernel<<<296, 256, 0, g->stream>>>(n_dev, a, g->np);
    CU(cudaGetLastError());
    g->launch_count += 1;
    int rc;
    if ((rc = launch_plane_fwd(g, 1, a, g->d_work))) return rc;
    if ((rc = launch_xpencil(g, 1, g->d_work, g->d_work, 3))) return rc;
    tdh::Epilogue ep;
    memset(&ep, 0, sizeof(ep));
    ep.alpha = make_double2(1.0, 0.0);
    ep.nx = g->n[0];
    if ((rc = launch_plane_inv(g, 1, g->d_work, nullptr, a, ep))) return rc;
    complex_to_real_kernel<<<296, 256, 0, g->stream>>>(a, vh_dev, g->np);
    CU(cudaGetLastError());
    g->launch_count += 1;
    return prof_collect(g);
}

// ------------------------------------------------------------------------------------------------------------
// NEXT-4: gradient in Fourier space and the forces of Eq. 11 (reading R20)
// ------------------------------------------------------------------------------------------------------------
// out = i (G_a + k_a) in on a spectrum in work layout [state][x][Y][z'] (x natural, Y and z' permuted: the tables are in
// the same orders)
__global__ void grad_scale_kernel(const cd* __restrict__ in, cd* __restrict__ out, size_t total, int nx, int ny, int nz,
                                  const double* __restrict__ gs, int axis) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int z = (int)(i % nz), y = (int)((i / nz) % ny), x = (int)((i / ((size_t)nz * ny)) % nx);
        const double ga = gs[axis == 0 ? x : (axis == 1 ? y : z)];
        const cd v = __ldcs(in + i);
        __stcs(out + i, make_double2(-ga * v.y, ga * v.x));
    }
}

// gd[p] (+)= sum_s occ[s] 2 Re( conj(grad_s[p]) psi_s[p] ), states in order
__global__ void grad_density_kernel(const cd* __restrict__ grad, const cd* __restrict__ psi, size_t npts, int nst,
                                    const double* __restrict__ occ, double* __restrict__ gd, int accumulate) {
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npts) return;
    double acc = accumulate ? gd[p] : 0.0;
    for (int s = 0; s < nst; ++s) {
        const cd a = __ldcs(grad + (size_t)s * npts + p), b = __ldcs(psi + (size_t)s * npts + p);
        acc += (occ ? occ[s] : 1.0) * 2.0 * (a.x * b.x + a.y * b.y);
    }
    gd[p] = acc;
}

// f[I][axis] += sum_s occ[s] 2 Re sum_{c in I} conj(dpig[s][c]) dpi[s][c]   (one thread per atom, fixed order)
__global__ void force_nl_kernel(const tdh::AtomDesc* __restrict__ atoms, int natoms, int nst, int nct, const cd* __restrict__ dpig,
                                const cd* __restrict__ dpi, const double* __restrict__ occ, int axis, double* __restrict__ f) {
    const int ia = blockIdx.x * blockDim.x + threadIdx.x;
    if (ia >= natoms) return;
    const tdh::AtomDesc at = atoms[ia];
    double acc = 0.0;
    for (int s = 0; s < nst; ++s) {
        double t = 0.0;
        for (int c = 0; c < at.nchan; ++c) {
            const cd a = dpig[(size_t)s * nct + at.chan0 + c], b = dpi[(size_t)s * nct + at.chan0 + c];
            t += a.x * b.x + a.y * b.y;
        }
        acc += (occ ? occ[s] : 1.0) * 2.0 * t;
    }
    f[3 * ia + axis] += acc;
}

// partial[(I*3 + a)*64 + slice] = sum over the slice's points of v_I[p] gd_a[p]; grid (64, natoms*3), 256 threads
__global__ void force_loc_partial_kernel(const double* __restrict__ vloc, const double* __restrict__ gd, size_t npts,
                                         double* __restrict__ partial) {
    __shared__ double red[8];
    const int ia = blockIdx.y / 3, a = blockIdx.y % 3, slice = blockIdx.x;
    const size_t per = (npts + 63) / 64, p0 = (size_t)slice * per, p1 = p0 + per < npts ? p0 + per : npts;
    const double* v = vloc + (size_t)ia * npts;
    const double* d = gd + (size_t)a * npts;
    double acc = 0.0;
    for (size_t p = p0 + threadIdx.x; p < p1; p += blockDim.x) acc += v[p] * d[p];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += red[w];
        partial[(size_t)blockIdx.y * 64 + slice] = t;
    }
}
__global__ void force_loc_final_kernel(const double* __restrict__ partial, int n3, double dv, double* __restrict__ f) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n3) return;
    double t = 0.0;
    for (int k = 0; k < 64; ++k) t += partial[(size_t)i * 64 + k];
    f[i] += dv * t;
}

// spectrum of a chunk in work layout into d_work (forward (z,y), forward x)
static int forward_spectrum(tdh_grid* g, int nst, const cd* in) {
    int rc;
    if ((rc = launch_plane_fwd(g, nst, in, g->d_work))) return rc;
    return launch_xpencil(g, nst, g->d_work, g->d_work, 1);
}
// out = d_axis of the states whose spectrum is in d_work; uses d_phi[1] as the second spectrum buffer
static int gradient_from_spectrum(tdh_grid* g, int nst, int axis, cd* out) {
    const size_t total = (size_t)nst * g->np;
    grad_scale_kernel<<<1184, 256, 0, g->stream>>>(g->d_work, g->d_phi[1], total, g->n[0], g->n[1], g->n[2], g->d_gs[axis], axis);
    CU(cudaGetLastError());
    g->launch_count += 1;
    int rc;
    if ((rc = launch_xpencil(g, nst, g->d_phi[1], g->d_phi[1], 2))) return rc;
    tdh::Epilogue ep;
    memset(&ep, 0, sizeof(ep));
    ep.alpha = make_double2(1.0, 0.0);
    ep.nx = g->n[0];
    return launch_plane_inv(g, nst, g->d_phi[1], nullptr, out, ep);
}

extern "C" int tdh_gradient(tdh_grid* g, int nst, const tdh_c128* psi_dev, int axis, tdh_c128* out_dev) {
    if (!g || !psi_dev || !out_dev) return fail(TDH_EINVAL, "tdh_gradient: null argument");
    NOT_SLAB("tdh_gradient");
    if (nst < 1 || nst > g->max_states) return fail(TDH_EINVAL, "tdh_gradient: nst = %d outside [1, %d]", nst, g->max_states);
    if (axis < 0 || axis > 2) return fail(TDH_EINVAL, "tdh_gradient: axis must be 0, 1 or 2");
    if (overlaps(psi_dev, out_dev, (size_t)nst * g->np * sizeof(cd))) return fail(TDH_EINVAL, "tdh_gradient: psi and out overlap");
    stats_reset(g);
    for (int s0 = 0; s0 < nst; s0 += g->chunk) {
        const int c = std::min(g->chunk, nst - s0);
        int rc;
        if ((rc = forward_spectrum(g, c, (const cd*)psi_dev + (size_t)s0 * g->np))) return rc;
        if ((rc = gradient_from_spectrum(g, c, axis, (cd*)out_dev + (size_t)s0 * g->np))) return rc;
    }
    return prof_collect(g);
}

extern "C" int tdh_forces(tdh_grid* g, int nst, const tdh_c128* psi_dev, const double* occ_host, const double* vloc_atoms_dev,
                          double* forces_host) {
    if (!g || !psi_dev || !forces_host) return fail(TDH_EINVAL, "tdh_forces: null argument");
    NOT_SLAB("tdh_forces");
    if (nst < 1 || nst > g->max_states) return fail(TDH_EINVAL, "tdh_forces: nst = %d outside [1, %d]", nst, g->max_states);
    if (g->natoms < 1) return fail(TDH_EINVAL, "tdh_forces: no atoms (tdh_set_projectors)");
    stats_reset(g);
    const double* occ = nullptr;
    if (occ_host) {
        CU(cudaMemcpyAsync(g->d_occ, occ_host, sizeof(double) * nst, cudaMemcpyHostToDevice, g->stream));
        CU(cudaStreamSynchronize(g->stream));
        occ = g->d_occ;
    }
    if (vloc_atoms_dev && !g->d_gd) CU(cudaMalloc(&g->d_gd, sizeof(double) * 3 * g->np));     // first use
    const int n3 = 3 * g->natoms;
    CU(cudaMemsetAsync(g->d_force, 0, sizeof(double) * n3, g->stream));
    cd* grad = g->d_phi[0];
    for (int s0 = 0; s0 < nst; s0 += g->chunk) {
        const int c = std::min(g->chunk, nst - s0);
        const cd* x = (const cd*)psi_dev + (size_t)s0 * g->np;
        int rc;
        if ((rc = launch_nl_project(g, c, x))) return rc;                               // D dV <beta|psi>
        if ((rc = forward_spectrum(g, c, x))) return rc;
        for (int a = 0; a < 3; ++a) {
            if ((rc = gradient_from_spectrum(g, c, a, grad))) return rc;
            if ((rc = launch_nl_project(g, c, grad, g->d_dvscale, g->d_dpig))) return rc;  // dV <beta|d_a psi>
            force_nl_kernel<<<(g->natoms + 63) / 64, 64, 0, g->stream>>>(g->d_atoms, g->natoms, c, g->nchan_tot, g->d_dpig,
                                                                          g->d_dpi, occ ? occ + s0 : nullptr, a, g->d_force);
            CU(cudaGetLastError());
            g->launch_count += 1;
            if (vloc_atoms_dev) {
                grad_density_kernel<<<(unsigned)((g->np + 255) / 256), 256, 0, g->stream>>>(
                    grad, x, g->np, c, occ ? occ + s0 : nullptr, g->d_gd + (size_t)a * g->np, s0 > 0 ? 1 : 0);
                CU(cudaGetLastError());
                g->launch_count += 1;
            }
        }
    }
    if (vloc_atoms_dev) {
        double* partial = g->d_force + n3;
        force_loc_partial_kernel<<<dim3(64, n3), 256, 0, g->stream>>>(vloc_atoms_dev, g->d_gd, g->np, partial);
        CU(cudaGetLastError());
        force_loc_final_kernel<<<(n3 + 127) / 128, 128, 0, g->stream>>>(partial, n3, g->dv, g->d_force);
        CU(cudaGetLastError());
        g->launch_count += 2;
    }
    CU(cudaMemcpyAsync(forces_host, g->d_force, sizeof(double) * n3, cudaMemcpyDeviceToHost, g->stream));
    CU(cudaStreamSynchronize(g->stream));
    return prof_collect(g);
}

// ------------------------------------------------------------------------------------------------------------
// NEXT-3: Teter-preconditioned steepest-descent update (reading R19)
// ------------------------------------------------------------------------------------------------------------
constexpr int SD_SLICES = 32;

// partial[(s*SD_SLICES + slice)*3 + {0,1,2}] = sums over the slice's points of |psi|^2, Re conj(psi) h, Re conj(psi) t.
// grid (SD_SLICES, nst), 256 threads; fixed summation order (thread-strided, warp shuffles, warps in order).
__global__ void sd_dots_kernel(const cd* __restrict__ psi, const cd* __restrict__ h, const cd* __restrict__ t, size_t npts,
                               double* __restrict__ partial) {
    __shared__ double red[8][3];
    const int s = blockIdx.y, slice = blockIdx.x;
    const size_t per = (npts + SD_SLICES - 1) / SD_SLICES, p0 = (size_t)slice * per, p1 = p0 + per < npts ? p0 + per : npts;
    const cd* a = psi + (size_t)s * npts;
    const cd* b = h + (size_t)s * npts;
    const cd* c = t + (size_t)s * npts;
    double nn = 0.0, eh = 0.0, et = 0.0;
    for (size_t p = p0 + threadIdx.x; p < p1; p += blockDim.x) {
        const cd x = __ldcs(a + p), y = __ldcs(b + p), z = __ldcs(c + p);
        nn += x.x * x.x + x.y * x.y;
        eh += x.x * y.x + x.y * y.y;
        et += x.x * z.x + x.y * z.y;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        nn += __shfl_xor_sync(0xffffffffu, nn, o);
        eh += __shfl_xor_sync(0xffffffffu, eh, o);
        et += __shfl_xor_sync(0xffffffffu, et, o);
    }
    if ((threadIdx.x & 31) == 0) { red[threadIdx.x >> 5][0] = nn; red[threadIdx.x >> 5][1] = eh; red[threadIdx.x >> 5][2] = et; }
    __syncthreads();
    if (threadIdx.x < 3) {
        double v = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) v += red[w][threadIdx.x];
        partial[((size_t)s * SD_SLICES + slice) * 3 + threadIdx.x] = v;
    }
}

// eps[s] = <psi|H psi>/<psi|psi>, ts[s] = <psi|T psi>/<psi|psi> from the slice sums, in slice order
__global__ void sd_finalize_kernel(const double* __restrict__ partial, int nst, double* __restrict__ eps, double* __restrict__ ts) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nst) return;
    double nn = 0.0, eh = 0.0, et = 0.0;
    for (int k = 0; k < SD_SLICES; ++k) {
        nn += partial[((size_t)s * SD_SLICES + k) * 3 + 0];
        eh += partial[((size_t)s * SD_SLICES + k) * 3 + 1];
        et += partial[((size_t)s * SD_SLICES + k) * 3 + 2];
    }
    eps[s] = eh / nn;
    ts[s] = et / nn;
}

// h <- h - eps[s] psi   (the residual)
__global__ void sd_residual_kernel(const cd* __restrict__ psi, cd* __restrict__ h, size_t npts, const double* __restrict__ eps) {
    const int s = blockIdx.y;
    const double e = eps[s];
    const cd* a = psi + (size_t)s * npts;
    cd* b = h + (size_t)s * npts;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < npts; p += (size_t)gridDim.x * blockDim.x) {
        const cd x = __ldcs(a + p);
        cd y = __ldcs(b + p);
        y.x -= e * x.x;
        y.y -= e * x.y;
        __stcs(b + p, y);
    }
}

extern "C" int tdh_sd_step(tdh_grid* g, int nst, tdh_c128* psi_dev, tdh_c128* work_dev, double lambda, double* eig_host) {
    if (!g || !psi_dev || !work_dev) return fail(TDH_EINVAL, "tdh_sd_step: null argument");
    NOT_SLAB("tdh_sd_step");
    if (nst < 1 || nst > g->max_states) return fail(TDH_EINVAL, "tdh_sd_step: nst = %d outside [1, %d]", nst, g->max_states);
    if (!std::isfinite(lambda)) return fail(TDH_EINVAL, "tdh_sd_step: bad lambda");
    if (overlaps(psi_dev, work_dev, (size_t)nst * g->np * sizeof(cd)))
        return fail(TDH_EINVAL, "tdh_sd_step: psi and work overlap");
    if (!g->d_sd) CU(cudaMalloc(&g->d_sd, sizeof(double) * (size_t)g->max_states * (2 + 3 * SD_SLICES)));   // first use
    stats_reset(g);
    double* eps = g->d_sd;
    double* ts = g->d_sd + g->max_states;
    double* partial = g->d_sd + 2 * (size_t)g->max_states;
    const cd one = make_double2(1.0, 0.0);
    for (int s0 = 0; s0 < nst; s0 += g->chunk) {
        const int c = std::min(g->chunk, nst - s0);
        cd* x = (cd*)psi_dev + (size_t)s0 * g->np;
        cd* h = (cd*)work_dev + (size_t)s0 * g->np;
        cd* t = g->d_phi[0];
        int rc;
        if ((rc = apply_chunk(g, c, x, h, one, nullptr))) return rc;                 // h = H psi
        if ((rc = apply_chunk(g, c, x, t, one, nullptr, true))) return rc;           // t = T psi
        sd_dots_kernel<<<dim3(SD_SLICES, c), 256, 0, g->stream>>>(x, h, t, g->np, partial);
        CU(cudaGetLastError());
        sd_finalize_kernel<<<(c + 127) / 128, 128, 0, g->stream>>>(partial, c, eps + s0, ts + s0);
        CU(cudaGetLastError());
        sd_residual_kernel<<<dim3(64, c), 256, 0, g->stream>>>(x, h, g->np, eps + s0);
        CU(cudaGetLastError());
        g->launch_count += 3;
        // psi <- psi - lambda K r : forward (z,y), x pass with the Teter factor, inverse (y,z) with the axpy epilogue
        if ((rc = launch_plane_fwd(g, c, h, g->d_work))) return rc;
        if ((rc = launch_xpencil(g, c, g->d_work, g->d_work, 4, ts + s0))) return rc;
        tdh::Epilogue ep;
        memset(&ep, 0, sizeof(ep));
        ep.yv = x;
        ep.alpha = make_double2(-lambda, 0.0);
        ep.nx = g->n[0];
        if ((rc = launch_plane_inv(g, c, g->d_work, nullptr, x, ep))) return rc;
    }
    if (eig_host) {
        CU(cudaMemcpyAsync(eig_host, eps, sizeof(double) * nst, cudaMemcpyDeviceToHost, g->stream));
        CU(cudaStreamSynchronize(g->stream));
    }
    return prof_collect(g);
}

// S = dV a^H b on FP64 tensor cores, split-K partials in the work buffer (overlap_kernels.cuh)
static int overlap_impl(tdh_grid* g, int na, const tdh_c128* a_dev, int nb, const tdh_c128* b_dev, tdh_c128* s_dev,
                        bool result_is_hermitian);

extern "C" int tdh_overlap(tdh_grid* g, int na, const tdh_c128* a_dev, int nb, const tdh_c128* b_dev, tdh_c128* s_dev) {
    return overlap_impl(g, na, a_dev, nb, b_dev, s_dev, false);
}

// result_is_hermitian: the caller knows that dV a^H b is Hermitian up to rounding (b = H a with a Hermitian H): only the
// tiles on and above the diagonal are computed, the others are their conjugate transposes (as for the Gram matrix)
static int overlap_impl(tdh_grid* g, int na, const tdh_c128* a_dev, int nb, const tdh_c128* b_dev, tdh_c128* s_dev,
                        bool result_is_hermitian) {
    if (!g || !a_dev || !b_dev || !s_dev) return fail(TDH_EINVAL, "tdh_overlap: null argument");
    if (na < 1 || nb < 1) return fail(TDH_EINVAL, "tdh_overlap: na, nb must be >= 1");
    stats_reset(g);
    const int ti = (na + tdh::OV_T - 1) / tdh::OV_T, tj = (nb + tdh::OV_T - 1) / tdh::OV_T;
    const size_t tile_cells = (size_t)ti * tj * tdh::OV_T * tdh::OV_T;
    const size_t cap = g->work_cells;                                      // complex values the work buffer holds
    if (tile_cells > cap) return fail(TDH_EUNSUPPORTED, "tdh_overlap: %d x %d does not fit the workspace", na, nb);
    const size_t nchunks = (g->np + tdh::OV_KC - 1) / tdh::OV_KC;
    // enough slices of K for about four waves of CTAs, bounded by the workspace and by 8 chunks per slice
    int dev = 0, nsm = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    size_t ksplit = std::max<size_t>(1, ((size_t)8 * nsm + (size_t)ti * tj - 1) / ((size_t)ti * tj));
    ksplit = std::min(ksplit, std::max<size_t>(1, nchunks / 8));
    ksplit = std::min(ksplit, cap / tile_cells);
    ksplit = std::min<size_t>(ksplit, 65535);
    int cps = (int)((nchunks + ksplit - 1) / ksplit);
    ksplit = (nchunks + cps - 1) / cps;
    size_t npts = g->np;
    int tjv = tj;
    cd* part = g->d_work;
    const cd* a = (const cd*)a_dev;
    const cd* b = (const cd*)b_dev;
    int hermitian = (na == nb && (a_dev == b_dev || result_is_hermitian)) ? 1 : 0;      // Gram matrix of one block: upper tiles only
    {
        void* args[] = {(void*)&a, (void*)&na, (void*)&b, (void*)&nb, (void*)&npts, (void*)&tjv, (void*)&cps, (void*)&part,
                        (void*)&hermitian};
        CU(cudaLaunchKernel(reinterpret_cast<const void*>(&tdh::overlap_kernel), dim3(ti * tj, (unsigned)ksplit),
                            dim3(tdh::OV_THREADS), args, 0, g->stream));
        g->launch_count += 1;
    }
    const int na_pad = ti * tdh::OV_T, nb_pad = tj * tdh::OV_T, ks = (int)ksplit;
    tdh::overlap_reduce_kernel<<<(na * nb + 255) / 256, 256, 0, g->stream>>>(part, ks, na, nb, na_pad, nb_pad, g->dv,
                                                                            (cd*)s_dev, hermitian);
    CU(cudaGetLastError());
    g->launch_count += 1;
    return TDH_OK;
}

static int launch_rotate(tdh_grid* g, int n_in, const cd* in, int n_out, const cd* m, cd* out, int upper) {
    size_t npts = g->np;
    void* args[] = {(void*)&in, (void*)&n_in, (void*)&m, (void*)&n_out, (void*)&npts, (void*)&upper, (void*)&out};
    dim3 grid((unsigned)((g->np + tdh::RT_P - 1) / tdh::RT_P), (n_out + tdh::RT_J - 1) / tdh::RT_J);
    CU(cudaLaunchKernel(reinterpret_cast<const void*>(&tdh::rotate_kernel), grid, dim3(tdh::OV_THREADS), args, 0, g->stream));
    g->launch_count += 1;
    return TDH_OK;
}

// out_j = sum_i psi_i m[i][j]: rotation in the space of states on FP64 tensor cores (overlap_kernels.cuh)
extern "C" int tdh_rotate(tdh_grid* g, int n_in, const tdh_c128* psi_dev, int n_out, const tdh_c128* m_dev,
                          tdh_c128* out_dev) {
    if (!g || !psi_dev || !m_dev || !out_dev) return fail(TDH_EINVAL, "tdh_rotate: null argument");
    if (n_in < 1 || n_out < 1 || n_out > 65535 * tdh::RT_J) return fail(TDH_EINVAL, "tdh_rotate: bad n_in / n_out");
    {
        const char* x = (const char*)psi_dev;
        const char* y = (const char*)out_dev;
        const size_t bx = (size_t)n_in * g->np * sizeof(cd), by = (size_t)n_out * g->np * sizeof(cd);
        if (x < y + by && y < x + bx) return fail(TDH_EINVAL, "tdh_rotate: psi and out overlap");
    }
    stats_reset(g);
    return launch_rotate(g, n_in, (const cd*)psi_dev, n_out, (const cd*)m_dev, (cd*)out_dev, 0);
}

// n x n scratch matrices of the rotations in the space of states: allocated at first use, grown for a larger block
static int small_scratch(tdh_grid* g, int nst) {
    if (g->small_n >= nst) return TDH_OK;
    CU(cudaStreamSynchronize(g->stream));
    for (int i = 0; i < 3; ++i) { cudaFree(g->d_small[i]); g->d_small[i] = nullptr; }
    cudaFree(g->d_w); g->d_w = nullptr;
    g->small_n = 0;
    for (int i = 0; i < 3; ++i) CU(cudaMalloc(&g->d_small[i], sizeof(cd) * (size_t)nst * nst));
    CU(cudaMalloc(&g->d_w, sizeof(double) * (size_t)nst));
    if (!g->d_status) CU(cudaMalloc(&g->d_status, 2 * sizeof(int)));       // [0] status, [1] grid-barrier counter
    if (!g->d_ctl) CU(cudaMalloc(&g->d_ctl, 8 * sizeof(unsigned)));
    g->small_n = nst;
    return TDH_OK;
}

// Subspace diagonalisation of an orthonormal block: M = dV psi^H (H psi) = V diag(w) V^H, out = psi V
extern "C" int tdh_subspace_diag(tdh_grid* g, int nst, const tdh_c128* psi_dev, const tdh_c128* hpsi_dev, tdh_c128* out_dev,
                                 double* eig_host) {
    if (!g || !psi_dev || !hpsi_dev || !out_dev) return fail(TDH_EINVAL, "tdh_subspace_diag: null argument");
    NOT_SLAB("tdh_subspace_diag");
    if (nst < 1 || nst > 1024) return fail(nst < 1 ? TDH_EINVAL : TDH_EUNSUPPORTED, "tdh_subspace_diag: nst = %d outside [1, 1024]", nst);
    if (overlaps(psi_dev, out_dev, (size_t)nst * g->np * sizeof(cd)))
        return fail(TDH_EINVAL, "tdh_subspace_diag: psi and out overlap");
    int rc = small_scratch(g, nst);
    if (rc) return rc;
    // M = dV psi^H (H psi) is Hermitian up to rounding: upper tiles only, then (M + M^H) / 2 inside the diagonal tiles
    if ((rc = overlap_impl(g, nst, psi_dev, nst, hpsi_dev, (tdh_c128*)g->d_small[1], true))) return rc;
    tdh::symmetrize_kernel<<<296, 256, 0, g->stream>>>(g->d_small[1], nst, g->d_small[0]);
    CU(cudaGetLastError());
    {
        int dev = 0, nsm = 0, occ = 0;
        CU(cudaGetDevice(&dev));
        CU(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
        const size_t smem = sizeof(tdh::JacobiRot) * (size_t)(nst / 2 + 1);
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, tdh::jacobi_eigh_kernel, tdh::JACOBI_T, smem));
        if (occ < 1) return fail(TDH_ECUDA, "tdh_subspace_diag: the eigensolver kernel does not fit on an SM");
        const size_t blocks = (size_t)(nst / 2 + 1) * (nst / 2 + 1) + (size_t)nst * (nst / 2 + 1);
        const int want = (int)((blocks + tdh::JACOBI_T - 1) / tdh::JACOBI_T);
        int per_sm = 1;                                                 // one CTA per SM: the grid barrier is the cost
        if (const char* e = getenv("TDH_JACOBI_CTAS_PER_SM")) per_sm = std::max(1, std::min(occ, atoi(e)));
        const int ctas = std::max(1, std::min(nsm * per_sm, want));
        CU(cudaMemsetAsync(g->d_ctl, 0, 8 * sizeof(unsigned), g->stream));
        cd* a = g->d_small[0];
        cd* a2 = g->d_small[2];
        cd* v = g->d_small[1];
        int n = nst;
        unsigned* ctl = g->d_ctl;
        void* args[] = {(void*)&a, (void*)&a2, (void*)&v, (void*)&n, (void*)&ctl};
        CU(cudaLaunchCooperativeKernel(reinterpret_cast<const void*>(&tdh::jacobi_eigh_kernel), dim3(ctas), dim3(tdh::JACOBI_T),
                                       args, smem, g->stream));
    }
    tdh::eigh_sort_kernel<<<1, 256, sizeof(double) * nst, g->stream>>>(g->d_small[0], g->d_small[1], nst, g->d_w, g->d_small[2]);
    CU(cudaGetLastError());
    g->launch_count += 3;
    if ((rc = launch_rotate(g, nst, (const cd*)psi_dev, nst, g->d_small[2], (cd*)out_dev, 0))) return rc;
    // the sweep count and the non-convergence flag come back with or without eig_host: an unconverged rotation must not
    // be returned as success
    unsigned ctl_host[8] = {0};
    if (eig_host) CU(cudaMemcpyAsync(eig_host, g->d_w, sizeof(double) * nst, cudaMemcpyDeviceToHost, g->stream));
    CU(cudaMemcpyAsync(ctl_host, g->d_ctl, sizeof(ctl_host), cudaMemcpyDeviceToHost, g->stream));
    CU(cudaStreamSynchronize(g->stream));
    g->jacobi_sweeps = (int)ctl_host[4];
    if (ctl_host[5] != 0)
        return fail(TDH_ECUDA, "tdh_subspace_diag: the Jacobi eigensolver did not converge in %u sweeps (non-finite input?); out is not a diagonalising rotation", ctl_host[4]);
    return TDH_OK;
}

// Cholesky orthonormalisation: S = dV psi^H psi = L L^H, out = psi L^{-H}
extern "C" int tdh_orthonormalize(tdh_grid* g, int nst, const tdh_c128* psi_dev, tdh_c128* out_dev) {
    if (!g || !psi_dev || !out_dev) return fail(TDH_EINVAL, "tdh_orthonormalize: null argument");
    NOT_SLAB("tdh_orthonormalize");
    if (nst < 1 || nst > 1024) return fail(nst < 1 ? TDH_EINVAL : TDH_EUNSUPPORTED, "tdh_orthonormalize: nst = %d outside [1, 1024]", nst);
    if (overlaps(psi_dev, out_dev, (size_t)nst * g->np * sizeof(cd)))
        return fail(TDH_EINVAL, "tdh_orthonormalize: psi and out overlap");
    int rc = small_scratch(g, nst);
    if (rc) return rc;
    rc = tdh_overlap(g, nst, psi_dev, nst, psi_dev, (tdh_c128*)g->d_small[0]);
    if (rc) return rc;
    {
        // cooperative launch: as many CTAs as are resident at once, at most one warp per row
        int dev = 0, nsm = 0, occ = 0;
        CU(cudaGetDevice(&dev));
        CU(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, tdh::cholesky_kernel, 256, 0));
        const int ctas = std::max(1, std::min(nsm * std::min(occ, 2), (nst + 7) / 8));
        CU(cudaMemsetAsync(g->d_status + 1, 0, sizeof(unsigned), g->stream));
        cd* sm = g->d_small[0];
        int n = nst;
        int* status = g->d_status;
        unsigned* barrier = reinterpret_cast<unsigned*>(g->d_status + 1);
        void* args[] = {(void*)&sm, (void*)&n, (void*)&status, (void*)&barrier};
        CU(cudaLaunchCooperativeKernel(reinterpret_cast<const void*>(&tdh::cholesky_kernel), dim3(ctas), dim3(256), args, 0,
                                       g->stream));
    }
    {
        const int warps = 4;
        const size_t smem = (size_t)warps * nst * sizeof(cd);
        CU(cudaFuncSetAttribute(tdh::inverse_lower_conjtrans_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        tdh::inverse_lower_conjtrans_kernel<<<(nst + warps - 1) / warps, 32 * warps, smem, g->stream>>>(g->d_small[0], nst,
                                                                                                     g->d_small[2]);
        CU(cudaGetLastError());
    }
    g->launch_count += 2;
    if ((rc = launch_rotate(g, nst, (const cd*)psi_dev, nst, g->d_small[2], (cd*)out_dev, 1))) return rc;
    int status = 0;
    CU(cudaMemcpyAsync(&status, g->d_status, sizeof(int), cudaMemcpyDeviceToHost, g->stream));
    CU(cudaStreamSynchronize(g->stream));
    if (status != 0) return fail(TDH_EINVAL, "tdh_orthonormalize: the states are linearly dependent (pivot %d of the overlap matrix is not positive)", status - 1);
    return TDH_OK;
}

extern "C" int tdh_fft3d(tdh_grid* g, int nst, tdh_c128* psi_dev, int sign) {
    if (!g || !psi_dev) return fail(TDH_EINVAL, "tdh_fft3d: null argument");
    NOT_SLAB("tdh_fft3d");
    if (nst < 1) return fail(TDH_EINVAL, "tdh_fft3d: nst < 1");
    if (sign != 1 && sign != -1) return fail(TDH_EINVAL, "tdh_fft3d: sign must be -1 or +1");
    stats_reset(g);
    cd* p = (cd*)psi_dev;
    // through the workspace, chunk by chunk (the tile kernels do not work in place when the planes are split)
    for (int s0 = 0; s0 < nst; s0 += g->chunk) {
        const int c = std::min(g->chunk, nst - s0);
        cd* q = p + (size_t)s0 * g->np;
        int rc;
        if (sign < 0) {
            if ((rc = launch_plane_fwd(g, c, q, g->d_work))) return rc;
            if ((rc = launch_xpencil(g, c, g->d_work, g->d_work, 1))) return rc;
            if ((rc = launch_reorder(g, c, g->d_work, q, 0))) return rc;
        } else {
            if ((rc = launch_reorder(g, c, q, g->d_work, 1))) return rc;
            if ((rc = launch_xpencil(g, c, g->d_work, g->d_work, 2))) return rc;
            tdh::Epilogue ep;
            memset(&ep, 0, sizeof(ep));
            ep.alpha = make_double2(1.0, 0.0);
            ep.nx = g->n[0];
            if ((rc = launch_plane_inv(g, c, g->d_work, nullptr, q, ep))) return rc;
        }
    }
    return prof_collect(g);
}

// ------------------------------------------------------------------------------------------------------------
// NEXT-4: slab decomposition of the grid over ranks (Fig. 6).  The all-to-all of the
// parallel 3-D transform is fused into the stores of the kernels that produce the data (tile_fwd: spectrum rows to
// their owners' Fourier-space slabs; xpencil: plane values to their owners' real-space work buffers), so a rank's
// Hamiltonian application is four stream-ordered phases with a cross-rank barrier between them and no copy kernels.
// ------------------------------------------------------------------------------------------------------------
// dpi[i] = sum over ranks (in rank order: every rank gets bitwise the same sum) of the partial projections
__global__ void slab_reduce_dpi_kernel(cd* __restrict__ dpi, size_t n, int world, const cd* p0, const cd* p1, const cd* p2,
                                       const cd* p3, const cd* p4, const cd* p5, const cd* p6, const cd* p7) {
    const cd* ps[8] = {p0, p1, p2, p3, p4, p5, p6, p7};
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        cd acc = make_double2(0.0, 0.0);
        for (int q = 0; q < world; ++q) {
            const cd v = __ldcg(ps[q] + i);
            acc.x += v.x;
            acc.y += v.y;
        }
        dpi[i] = acc;
    }
}

extern "C" int tdh_slab_buffers(tdh_grid* g, void** fs_dev, void** rs_dev, void** dpi_dev) {
    if (!g) return fail(TDH_EINVAL, "tdh_slab_buffers: null handle");
    if (g->slab_world < 2) return fail(TDH_EINVAL, "tdh_slab_buffers: not a slab handle");
    if (fs_dev) *fs_dev = g->d_fs;
    if (rs_dev) *rs_dev = g->d_work;
    if (dpi_dev) *dpi_dev = g->d_dpi_part;
    return TDH_OK;
}

extern "C" int tdh_slab_set_peers(tdh_grid* g, void* const* fs_dev, void* const* rs_dev, void* const* dpi_dev) {
    if (!g || !fs_dev || !rs_dev) return fail(TDH_EINVAL, "tdh_slab_set_peers: null argument");
    if (g->slab_world < 2) return fail(TDH_EINVAL, "tdh_slab_set_peers: not a slab handle");
    for (int q = 0; q < g->slab_world; ++q) {
        if (!fs_dev[q] || !rs_dev[q]) return fail(TDH_EINVAL, "tdh_slab_set_peers: null buffer of rank %d", q);
        if (g->natoms > 0 && (!dpi_dev || !dpi_dev[q])) return fail(TDH_EINVAL, "tdh_slab_set_peers: projectors are set but rank %d has no projection buffer", q);
    }
    if (fs_dev[g->slab_rank] != g->d_fs || rs_dev[g->slab_rank] != g->d_work)
        return fail(TDH_EINVAL, "tdh_slab_set_peers: entry %d must be this handle's own buffers (tdh_slab_buffers)", g->slab_rank);
    CU(cudaStreamSynchronize(g->stream));
    for (int q = 0; q < g->slab_world; ++q) {
        g->peer_fs[q] = (cd*)fs_dev[q];
        g->peer_rs[q] = (cd*)rs_dev[q];
        g->peer_dpi[q] = dpi_dev ? (const cd*)dpi_dev[q] : nullptr;
    }
    g->have_peers = true;
    return TDH_OK;
}

static int slab_check(tdh_grid* g, const char* name, int nst) {
    if (!g) return fail(TDH_EINVAL, "%s: null handle", name);
    if (g->slab_world < 2) return fail(TDH_EINVAL, "%s: not a slab handle (tdh_create_slab_grid)", name);
    if (!g->have_peers) return fail(TDH_EINVAL, "%s: tdh_slab_set_peers has not been called", name);
    if (nst < 1 || nst > max_chunk(g)) return fail(TDH_EINVAL, "%s: nst = %d outside [1, %d] (one chunk per call)", name, nst, max_chunk(g));
    return TDH_OK;
}

extern "C" int tdh_slab_apply_phase(tdh_grid* g, int phase, int nst, const tdh_c128* psi_dev, tdh_c128* hpsi_dev) {
    int rc = slab_check(g, "tdh_slab_apply_phase", nst);
    if (rc) return rc;
    if (!psi_dev) return fail(TDH_EINVAL, "tdh_slab_apply_phase: null psi");
    const cd* in = (const cd*)psi_dev;
    if (phase == 0) stats_reset(g);
    switch (phase) {
        case TDH_SLAB_PROJECT:                      // partial projections over this rank's planes
            if (g->natoms > 0 && (rc = launch_nl_project(g, nst, in))) return rc;
            return TDH_OK;
        case TDH_SLAB_PLANES_FWD: {                 // sum of the ranks' projections; (z,y) transform, rows to their owners
            if (g->natoms > 0) {
                for (int q = 0; q < g->slab_world; ++q)
                    if (!g->peer_dpi[q]) return fail(TDH_EINVAL, "tdh_slab_apply_phase: projection buffer of rank %d not set", q);
                const size_t n = (size_t)nst * g->nchan_tot;
                const cd** pp = g->peer_dpi;
                slab_reduce_dpi_kernel<<<(unsigned)std::min<size_t>(296, (n + 255) / 256), 256, 0, g->stream>>>(
                    g->d_dpi, n, g->slab_world, pp[0], pp[1], pp[2], pp[3], pp[4], pp[5], pp[6], pp[7]);
                CU(cudaGetLastError());
                g->launch_count += 1;
            }
            return launch_plane_fwd(g, nst, in, nullptr, true);
        }
        case TDH_SLAB_PENCILS:                      // x transform, kinetic factor, inverse x: plane values to their owners
            return launch_xpencil(g, nst, g->d_fs, nullptr, 0, nullptr, true);
        case TDH_SLAB_PLANES_INV:                   // inverse (y,z) transform + epilogue on this rank's planes
            if (!hpsi_dev) return fail(TDH_EINVAL, "tdh_slab_apply_phase: null hpsi");
            if (overlaps(psi_dev, hpsi_dev, (size_t)nst * g->np * sizeof(cd)))
                return fail(TDH_EINVAL, "tdh_slab_apply_phase: psi and hpsi overlap");
            if ((rc = finish_chunk(g, nst, in, (cd*)hpsi_dev, make_double2(1.0, 0.0), nullptr))) return rc;
            return prof_collect(g);
        default:
            return fail(TDH_EINVAL, "tdh_slab_apply_phase: phase %d", phase);
    }
}

extern "C" int tdh_slab_fft_phase(tdh_grid* g, int sign, int phase, int nst, tdh_c128* block_dev) {
    int rc = slab_check(g, "tdh_slab_fft_phase", nst);
    if (rc) return rc;
    if (!block_dev) return fail(TDH_EINVAL, "tdh_slab_fft_phase: null block");
    if (sign != 1 && sign != -1) return fail(TDH_EINVAL, "tdh_slab_fft_phase: sign must be -1 or +1");
    if (phase != 0 && phase != 1) return fail(TDH_EINVAL, "tdh_slab_fft_phase: phase %d", phase);
    cd* blk = (cd*)block_dev;
    if (phase == 0) stats_reset(g);
    if (sign < 0) {
        if (phase == 0) return launch_plane_fwd(g, nst, blk, nullptr, true);            // real-space slab -> owners' rows
        return launch_xpencil(g, nst, g->d_fs, blk, 1);                                  // spectrum slab, work layout
    }
    if (phase == 0) return launch_xpencil(g, nst, blk, nullptr, 2, nullptr, true);      // spectrum slab -> owners' planes
    tdh::Epilogue ep;
    memset(&ep, 0, sizeof(ep));
    ep.alpha = make_double2(1.0, 0.0);
    ep.nx = g->n[0];
    return launch_plane_inv(g, nst, g->d_work, nullptr, blk, ep);
}

// CUDA IPC wrappers so that one process per GPU can hand its exchange buffers to its peers (shard.SlabRank)
extern "C" int tdh_ipc_export(void* dev_ptr, unsigned char handle[64]) {
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "IPC handle size");
    if (!dev_ptr || !handle) return fail(TDH_EINVAL, "tdh_ipc_export: null argument");
    cudaIpcMemHandle_t h;
    CU(cudaIpcGetMemHandle(&h, dev_ptr));
    memcpy(handle, &h, 64);
    return TDH_OK;
}
extern "C" int tdh_ipc_import(const unsigned char handle[64], void** dev_ptr) {
    if (!handle || !dev_ptr) return fail(TDH_EINVAL, "tdh_ipc_import: null argument");
    cudaIpcMemHandle_t h;
    memcpy(&h, handle, 64);
    CU(cudaIpcOpenMemHandle(dev_ptr, h, cudaIpcMemLazyEnablePeerAccess));
    return TDH_OK;
}
extern "C" int tdh_ipc_close(void* dev_ptr) {
    if (!dev_ptr) return TDH_OK;
    CU(cudaIpcCloseMemHandle(dev_ptr));
    return TDH_OK;
}

extern "C" int tdh_work_layout(const tdh_grid* g, int* rowmap_host, int* colmap_host) {
    if (!g || !rowmap_host || !colmap_host) return fail(TDH_EINVAL, "tdh_work_layout: null argument");
    CU(cudaMemcpy(rowmap_host, g->d_rowmap, sizeof(int) * g->n[1], cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(colmap_host, g->d_colmap, sizeof(int) * g->n[2], cudaMemcpyDeviceToHost));
    return TDH_OK;
}

// ------------------------------------------------------------------------------------------------------------
// host-buffer entry points: chunked, double-buffered H2D -> kernels -> D2H on three streams
// ------------------------------------------------------------------------------------------------------------
static int host_path_init(tdh_grid* g) {
    if (g->d_hin[0]) return TDH_OK;
    g->host_chunk = g->chunk_cap;
    // bound the four staging buffers to 512 MiB each
    const size_t state_bytes = g->np * sizeof(cd);
    g->host_chunk = (int)std::max<size_t>(1, std::min<size_t>((size_t)g->host_chunk, ((size_t)512 << 20) / state_bytes));
    for (int i = 0; i < 2; ++i) {
        CU(cudaMalloc(&g->d_hin[i], state_bytes * g->host_chunk));
        CU(cudaMalloc(&g->d_hout[i], state_bytes * g->host_chunk));
        CU(cudaEventCreateWithFlags(&g->ev_in[i], cudaEventDisableTiming));
        CU(cudaEventCreateWithFlags(&g->ev_k[i], cudaEventDisableTiming));
        CU(cudaEventCreateWithFlags(&g->ev_out[i], cudaEventDisableTiming));
    }
    CU(cudaStreamCreateWithFlags(&g->s_h2d, cudaStreamNonBlocking));
    CU(cudaStreamCreateWithFlags(&g->s_d2h, cudaStreamNonBlocking));
    return TDH_OK;
}

static int host_pipeline(tdh_grid* g, int nst, const cd* in_host, cd* out_host, bool propagate, double dt, int nsteps) {
    int rc = host_path_init(g);
    if (rc) return rc;
    stats_reset(g);
    const size_t state_bytes = g->np * sizeof(cd);
    const int hc = g->host_chunk;
    int it = 0;
    for (int s0 = 0; s0 < nst; s0 += hc, ++it) {
        const int c = std::min(hc, nst - s0);
        const int slot = it & 1;
        const size_t off = (size_t)s0 * g->np;
        // H2D into d_hin[slot] once the kernels (apply) or the D2H (propagate) that last used it are done
        if (it >= 2) CU(cudaStreamWaitEvent(g->s_h2d, propagate ? g->ev_out[slot] : g->ev_k[slot], 0));
        CU(cudaMemcpyAsync(g->d_hin[slot], in_host + off, state_bytes * c, cudaMemcpyHostToDevice, g->s_h2d));
        CU(cudaEventRecord(g->ev_in[slot], g->s_h2d));
        CU(cudaStreamWaitEvent(g->stream, g->ev_in[slot], 0));
        if (propagate) {
            if ((rc = propagate_block(g, c, g->d_hin[slot], dt, nsteps))) return rc;
        } else {
            if (it >= 2) CU(cudaStreamWaitEvent(g->stream, g->ev_out[slot], 0));
            if ((rc = apply_block(g, c, g->d_hin[slot], g->d_hout[slot]))) return rc;
        }
        CU(cudaEventRecord(g->ev_k[slot], g->stream));
        CU(cudaStreamWaitEvent(g->s_d2h, g->ev_k[slot], 0));
        CU(cudaMemcpyAsync(out_host + off, propagate ? g->d_hin[slot] : g->d_hout[slot], state_bytes * c,
                           cudaMemcpyDeviceToHost, g->s_d2h));
        CU(cudaEventRecord(g->ev_out[slot], g->s_d2h));
    }
    CU(cudaStreamSynchronize(g->s_h2d));
    CU(cudaStreamSynchronize(g->stream));
    CU(cudaStreamSynchronize(g->s_d2h));
    return prof_collect(g);
}

extern "C" int tdh_apply_hamiltonian_host(tdh_grid* g, int nst, const tdh_c128* psi_host, tdh_c128* hpsi_host) {
    if (!g || !psi_host || !hpsi_host) return fail(TDH_EINVAL, "tdh_apply_hamiltonian_host: null argument");
    NOT_SLAB("tdh_apply_hamiltonian_host");
    if (nst < 1) return fail(TDH_EINVAL, "tdh_apply_hamiltonian_host: nst < 1");
    if (overlaps(psi_host, hpsi_host, (size_t)nst * g->np * sizeof(cd)))
        return fail(TDH_EINVAL, "tdh_apply_hamiltonian_host: psi and hpsi overlap");
    return host_pipeline(g, nst, (const cd*)psi_host, (cd*)hpsi_host, false, 0.0, 0);
}

extern "C" int tdh_propagate_host(tdh_grid* g, int nst, tdh_c128* psi_host, double dt, int nsteps, int order) {
    if (!g || !psi_host) return fail(TDH_EINVAL, "tdh_propagate_host: null argument");
    NOT_SLAB("tdh_propagate_host");
    if (nst < 1) return fail(TDH_EINVAL, "tdh_propagate_host: nst < 1");
    if (order != 4) return fail(TDH_EINVAL, "tdh_propagate_host: order must be 4");
    if (nsteps < 0 || !std::isfinite(dt)) return fail(TDH_EINVAL, "tdh_propagate_host: bad dt / nsteps");
    return host_pipeline(g, nst, (const cd*)psi_host, (cd*)psi_host, true, dt, nsteps);
}

// ------------------------------------------------------------------------------------------------------------
// statistics / knobs
// ------------------------------------------------------------------------------------------------------------
extern "C" int tdh_last_launch_count(const tdh_grid* g) { return g ? g->launch_count : 0; }
extern "C" int tdh_last_jacobi_sweeps(const tdh_grid* g) { return g ? g->jacobi_sweeps : 0; }

extern "C" int tdh_set_profiling(tdh_grid* g, int on) {
    if (!g) return fail(TDH_EINVAL, "tdh_set_profiling: null handle");
    g->profiling = on != 0;
    g->epoch += 1;
    return TDH_OK;
}

extern "C" int tdh_last_kernel_seconds(const tdh_grid* g, double out[TDH_NKERNELS]) {
    if (!g || !out) return fail(TDH_EINVAL, "tdh_last_kernel_seconds: null argument");
    for (int i = 0; i < TDH_NKERNELS; ++i) out[i] = g->ksec[i];
    return TDH_OK;
}

extern "C" const char* tdh_kernel_name(int i) { return (i >= 0 && i < TDH_NKERNELS) ? kKernelNames[i] : ""; }

// Everything the calls below would otherwise allocate at their first use, allocated now (no allocation on
// hot paths): the n x n scratch of the rotations for blocks of up to rotation_states states, the per-state reduction
// scratch of tdh_sd_step, the gradient-density arrays of tdh_forces' local term, the staging buffers of the host entry points
extern "C" int tdh_reserve(tdh_grid* g, int rotation_states, int forces_local_term, int host_buffers) {
    if (!g) return fail(TDH_EINVAL, "tdh_reserve: null handle");
    if (rotation_states < 0 || rotation_states > g->max_states)
        return fail(TDH_EINVAL, "tdh_reserve: rotation_states = %d outside [0, %d]", rotation_states, g->max_states);
    int rc;
    if (rotation_states > 0 && (rc = small_scratch(g, rotation_states))) return rc;
    if (!g->d_sd) CU(cudaMalloc(&g->d_sd, sizeof(double) * (size_t)g->max_states * (2 + 3 * SD_SLICES)));
    if (forces_local_term && !g->d_gd) CU(cudaMalloc(&g->d_gd, sizeof(double) * 3 * g->np));
    if (host_buffers && g->slab_world == 1 && (rc = host_path_init(g))) return rc;
    return TDH_OK;
}

extern "C" int tdh_set_chunk_states(tdh_grid* g, int chunk) {
    if (!g) return fail(TDH_EINVAL, "tdh_set_chunk_states: null handle");
    if (chunk < 0) return fail(TDH_EINVAL, "tdh_set_chunk_states: chunk < 0");
    g->chunk = chunk == 0 ? default_chunk(g) : std::min(chunk, max_chunk(g));
    g->epoch += 1;
    return TDH_OK;
}

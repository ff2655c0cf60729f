/*
 * tdh.h -- C ABI of the B200-native Kohn-Sham H|psi> / Taylor-4 real-time TDDFT library (libtdh.so).
 *
 * The operation is the one the paper states as an operator applied to a field set, returning a field set:
 *     auto hphi = hamiltonian(phi);                                   PAPER.md:225 (section V)
 *     "a routine that applies the Hamiltonian over a field set"       PAPER.md:478 (section VIII.E)
 * with the field set one contiguous array holding all states          PAPER.md:466 (section VIII.D).
 *
 *     H psi = -1/2 nabla^2 psi + V(r) psi + V_nl psi                   Eq. 2
 *       kinetic term in Fourier space (diagonal, 1/2 |G+k|^2), via two batched 3-D FFTs
 *       local potential: pointwise product in real space
 *       non-local Kleinman-Bylander projectors on spheres in real space                     Eq. 9
 *     exp(-i dt H) psi ~= sum_{k=0..4} (-i dt)^k / k! H^k psi          Eq. 8
 *     ETRS step from two such sums sharing H^k psi                       Eq. 6-7
 *     n(r) = sum_s f_s |psi_s(r)|^2;  v_H from the periodic Poisson equation in Fourier space   Eq. 1
 *
 * Conventions (readings R1-R16 of DESIGN.md): orthorhombic periodic cell, atomic units (Hartree, bohr).
 * Grid point (i,j,k) sits at r = (i h_x, j h_y, k h_z), h_a = len[a]/n[a]; flat index p = (i*n[1] + j)*n[2] + k.
 *
 * LAYOUT.  A state block is psi[s][ix][iy][iz], iz fastest, state slowest, complex128 with interleaved (re, im):
 * exactly a contiguous torch tensor of shape (nst, n0, n1, n2), dtype complex128.  A sub-block of states is a
 * contiguous slice.  All internal layouts are the library's business.
 *
 * MEMORY SPACES.  Every pointer argument says DEVICE or HOST.  Device pointers must belong to the CUDA device that
 * was current when tdh_create_grid was called.
 *
 * OWNERSHIP.  The caller owns psi / hpsi.  The handle owns copies of V, of the projector tables, the FFT tables and
 * all workspace; everything is allocated in tdh_create_grid / tdh_set_*; tdh_apply_hamiltonian and tdh_propagate
 * allocate nothing (no allocation on hot paths).
 *
 * ASYNCHRONY.  tdh_apply_hamiltonian / tdh_propagate enqueue work on the handle's stream and return; the caller
 * synchronises the stream.  tdh_set_* and the *_host calls synchronise internally.
 *
 * ERRORS.  Every call returns 0 on success or a negative code; nothing throws or exits across this boundary.
 * tdh_last_error() returns a thread-local, statically stored message for the last failing call of this thread.
 *
 * ENVIRONMENT.  Read when a handle is created (TDH_NL_MODE, TDH_SCATTER_BULK: when projectors are set); all optional, the
 * defaults are the measured-best choices, the variables exist so that tests and profiles can run every path:
 *   TDH_SMALL=0             16^3 / 32^3 grids through the tiled kernels instead of the one-launch on-chip kernel
 *   TDH_SMALL16_CLUSTER=0   16^3 blocks of few states with one CTA per state instead of a cluster of four
 *   TDH_NL_MODE=0|1         back-projection as record lists inside the inverse transform (0) or as its own kernel (1)
 *   TDH_SCATTER_BULK=0|1    that kernel by load-add-store (0) or by bulk reduce-add in the L2 (1)
 *   TDH_GRAPH=0             tdh_propagate always as plain launches
 *   TDH_CHUNK_STATES=n, TDH_WORKSPACE_MB=m, TDH_MAX_CTAS_PER_SM=c, TDH_JACOBI_CTAS_PER_SM=c
 *                           states per launch, workspace per buffer (default 4096), persistent-grid sizes
 *
 * There is no CPU fallback anywhere in this library.
 */
#ifndef TDH_H
#define TDH_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tdh_grid tdh_grid;                 /* opaque handle */
typedef struct { double re, im; } tdh_c128;      /* one complex128 value */

enum {
    TDH_OK = 0,
    TDH_EINVAL = -1,        /* null pointer, nst < 1, nst > max_states, overlapping in/out, order != 4, ...       */
    TDH_EUNSUPPORTED = -2,  /* grid size not supported: every n[a] must be 2^a 3^b with 4 <= n[a] <= 256; a size limit
                               of one entry point (stated there)                                                   */
    TDH_ENOMEM = -3,        /* host or device allocation failed                                                   */
    TDH_ECUDA = -4,         /* CUDA runtime error (text in tdh_last_error)                                        */
    TDH_EINDEX = -5         /* sph_idx entry outside [0, n0*n1*n2), or a grid point listed twice for one atom     */
};

/* Create a grid handle.
 *   n[3]        HOST  grid points per axis; each must be 2^a 3^b with 4 <= n[a] <= 256 (else TDH_EUNSUPPORTED: a prime
 *                     factor other than 2 or 3, n[a] < 4, or n[a] > 256).  Grids whose three lengths all lie in
 *                     {16, 32, 48, 64, 96} (the BASELINE configs and their mixes) run the tuned TMA kernels; any other
 *                     grid runs the general shared-memory Stockham path (five launches per application, same results)
 *   len[3]      HOST  cell lengths in bohr, > 0
 *   kpt[3]      HOST  Bloch vector k, Cartesian, 1/bohr (reading R1: psi is the periodic part u_k; kinetic 1/2|G+k|^2)
 *   ecut              plane-wave cutoff in Ha for the kinetic term: components with 1/2|G+k|^2 > ecut are zeroed in
 *                     the kinetic term only (reading R6); ecut <= 0 or +inf means no mask
 *   max_states        largest nst any later call will pass (sizes the workspace), >= 1
 *   cuda_stream       a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream) or NULL for the default stream
 *   out               receives the handle
 * Initial state: V = 0, no projectors. */
int tdh_create_grid(const int n[3], const double len[3], const double kpt[3], double ecut, int max_states,
                    void* cuda_stream, tdh_grid** out);

/* Free everything the handle owns.  NULL is accepted. */
int tdh_destroy_grid(tdh_grid* g);

/* Set the local potential V(r) (sum of v_loc + v_H + v_xc of Eq. 2; "a simple multiplicative
 * potential").   v_dev: DEVICE, n0*n1*n2 doubles in grid layout; copied.  NULL resets V to 0. */
int tdh_set_potential(tdh_grid* g, const double* v_dev);

/* Set the Kleinman-Bylander projectors (Eq. 9; readings R2-R5).  All pointers are HOST; the
 * tables are copied and re-indexed internally.  natoms = 0 clears the projectors (other pointers may be NULL).
 *   sph_off   [natoms+1]   prefix sums of P_I (points in atom I's sphere), sph_off[0] = 0
 *   sph_idx   [sum P_I]    flat grid index p of each sphere point; within one atom every p at most once
 *   sph_disp  [sum P_I][3] minimum-image displacement r_p - R_I (bohr); used only for the Bloch phases
 *                          e^{+-i k.d} when k != 0; may be NULL when k = 0
 *   chan_off  [natoms+1]   prefix sums of C_I (projector channels of atom I), chan_off[0] = 0
 *   beta      concatenated per atom: [C_I][P_I] real projector values beta_{I,c}(r_q - R_I)
 *   dcoef     [sum C_I]    KB coefficients D_{I,c}
 * Computes  (V_nl psi)[S_I[q]] += e^{-ik.d_q} sum_c beta_{I,c}[q] D_{I,c} dV sum_{q'} beta_{I,c}[q'] e^{+ik.d_q'} psi[S_I[q']]. */
int tdh_set_projectors(tdh_grid* g, int natoms, const int64_t* sph_off, const int32_t* sph_idx,
                       const double* sph_disp, const int32_t* chan_off, const double* beta, const double* dcoef);

/* hpsi = H psi for a block of nst states (Eq. 2).  psi_dev, hpsi_dev: DEVICE, nst*n0*n1*n2 complex128 each, must not
 * overlap.  1 <= nst <= max_states.  Asynchronous on the handle's stream. */
int tdh_apply_hamiltonian(tdh_grid* g, int nst, const tdh_c128* psi_dev, tdh_c128* hpsi_dev);

/* nsteps steps of psi <- sum_{k=0..4} (-i dt)^k/k! H^k psi (Eq. 8 with lambda = -i dt; fixed H, reading R10), in place.
 * psi_dev: DEVICE, nst*n0*n1*n2 complex128.  order must be 4.  nsteps >= 0.  Asynchronous on the handle's stream.
 * Blocks of at most 128 MiB (the launch-latency regime) are replayed as one CUDA graph: the first call with a given
 * (psi_dev, nst, dt, nsteps) captures the call's launches on an internal stream and instantiates the graph (host work
 * only, nothing is allocated on the device), later calls with the same arguments launch that graph on the handle's
 * stream; any tdh_set_* call captures anew, and the handle keeps the graphs of the last four (buffer, count)
 * combinations.  The result is bitwise that of the plain
 * launches.  TDH_GRAPH=0 in the environment at tdh_create_grid switches the graph off. */
int tdh_propagate(tdh_grid* g, int nst, tdh_c128* psi_dev, double dt, int nsteps, int order);

/* The two exponentials of an ETRS step that share their powers H^k psi (Eq. 8 for two lambdas):
 *     full <- sum_{k=0..4} (-i dt)^k/k!   H^k psi        (Eq. 7: the approximate psi(t+dt) from which H(t+dt) is built)
 *     psi  <- sum_{k=0..4} (-i dt/2)^k/k! H^k psi        (the first factor of Eq. 6), in place
 * from four H applications instead of eight.  psi_dev, full_dev: DEVICE, nst*n0*n1*n2 complex128 each, must not overlap.
 * order must be 4.  Asynchronous on the handle's stream; allocates nothing. */
int tdh_taylor_pair(tdh_grid* g, int nst, tdh_c128* psi_dev, tdh_c128* full_dev, double dt, int order);

/* One ETRS step, Eq. 6-7, with the local potential at t+dt supplied by the caller:
 *     approx <- exp(-i dt H(t)) psi;   psi <- exp(-i dt/2 H(t+dt)) exp(-i dt/2 H(t)) psi      (Taylor order 4 each)
 * H(t) uses the handle's current potential, H(t+dt) uses v_next_dev (DEVICE, n0*n1*n2 doubles, or NULL for V = 0),
 * which becomes the handle's potential (as after tdh_set_potential); the projectors are the same in both.  This is
 * tdh_taylor_pair, a potential switch and tdh_propagate(dt/2, 1 step): 8 H applications.  When V(t+dt) has to be
 * derived from approx (self-consistent propagation), call those three yourself with your update in between.
 * approx_dev: DEVICE work/output block of the size of psi_dev, must not overlap it. */
int tdh_etrs_step(tdh_grid* g, int nst, tdh_c128* psi_dev, tdh_c128* approx_dev, double dt, const double* v_next_dev);

/* Density, Eq. 1:  n[p] = sum_s occ[s] |psi_s[p]|^2  over the nst states of the block ("a parallel
 * reduction over states"; with states sharded over GPUs the caller all-reduces n_dev afterwards).
 *   psi_dev   DEVICE  nst*n0*n1*n2 complex128         occ_host  HOST [nst] occupations, or NULL for all 1
 *   n_dev     DEVICE  n0*n1*n2 doubles                accumulate != 0: added to n_dev (blocks processed in pieces)
 * States are summed in order (deterministic).  Asynchronous on the handle's stream (synchronises once if occ_host). */
int tdh_density(tdh_grid* g, int nst, const tdh_c128* psi_dev, const double* occ_host, double* n_dev, int accumulate);

/* Hartree potential of a periodic density (the Poisson equation solved in Fourier space):
 *   v_hat(G) = 4 pi n_hat(G) / |G|^2 for G != 0, v_hat(0) = 0;  periodic boundary conditions only.
 * n_dev, vh_dev: DEVICE, n0*n1*n2 doubles each (may be the same array).  Uses the handle's workspace: do not run
 * concurrently with other calls on the same handle.  Asynchronous on the handle's stream. */
int tdh_hartree(tdh_grid* g, const double* n_dev, double* vh_dev);

/* Overlap / subspace matrix of two state blocks (first building block of the ground-state rotations, PAPER.md:393;
 * also the check that propagation keeps the states orthonormal):
 *     S[i][j] = dV sum_p conj(a_i[p]) b_j[p],   i < na, j < nb,   row-major [na][nb] complex128
 * a_dev, b_dev: DEVICE blocks of na / nb states (may be the same block); s_dev: DEVICE, na*nb complex128.
 * A flop-bound complex GEMM on FP64 tensor cores, split over K with a deterministic reduction.  Uses the handle's
 * workspace (na, nb rounded up to 64 must satisfy na*nb <= workspace / 16 bytes).  Any grid the handle accepts (the
 * last chunk of K, and the last tile of points of tdh_rotate, are predicated).  Asynchronous on the handle's stream. */
int tdh_overlap(tdh_grid* g, int na, const tdh_c128* a_dev, int nb, const tdh_c128* b_dev, tdh_c128* s_dev);

/* Rotation in the space of states ("rotations in the space of eigenvectors"):
 *     out_j[p] = sum_i psi_i[p] m[i][j],   i < n_in, j < n_out
 * psi_dev: DEVICE block of n_in states; m_dev: DEVICE, row-major [n_in][n_out] complex128; out_dev: DEVICE block of
 * n_out states, must not overlap psi_dev.  A flop-bound complex GEMM on FP64 tensor cores.  Asynchronous. */
int tdh_rotate(tdh_grid* g, int n_in, const tdh_c128* psi_dev, int n_out, const tdh_c128* m_dev, tdh_c128* out_dev);

/* Cholesky orthonormalisation ("orthogonalization"): S = dV psi^H psi = L L^H, out = psi L^{-H}, so that
 * dV out^H out = 1 and out_j mixes psi_0..psi_j only (the Gram-Schmidt order).  tdh_overlap, a cooperative Cholesky and
 * a triangular inverse of the nst x nst matrix, tdh_rotate.  1 <= nst <= 1024; psi_dev, out_dev: DEVICE blocks of nst
 * states, must not overlap.  The first call (or a larger nst) allocates two nst x nst scratch matrices.
 * Synchronises the stream; returns TDH_EINVAL when the states are linearly dependent (out is then undefined). */
int tdh_orthonormalize(tdh_grid* g, int nst, const tdh_c128* psi_dev, tdh_c128* out_dev);

/* Subspace diagonalisation of an ORTHONORMAL block: M = dV psi^H (H psi) = V diag(w) V^H, out = psi V,
 * so that dV out^H H out = diag(w), w ascending.  hpsi_dev holds H psi (tdh_apply_hamiltonian).  tdh_overlap, a
 * cooperative parallel Jacobi eigensolver of the nst x nst Hermitian matrix, tdh_rotate.  1 <= nst <= 1024.
 * psi_dev, hpsi_dev, out_dev: DEVICE blocks of nst states, out must not overlap psi; eig_host: HOST [nst] or NULL.
 * hpsi_dev must be a HERMITIAN operator applied to psi_dev (what tdh_apply_hamiltonian returns): only the tiles of M on
 * and above the diagonal are computed and the others are taken as their conjugate transposes; for any other hpsi the
 * result is the diagonalisation of that mirrored matrix, not of (M + M^H)/2.  Synchronises the stream (the sweep count
 * and the convergence flag of the eigensolver are read back): TDH_ECUDA when the Jacobi iteration has not converged in
 * 40 sweeps (non-finite input), out is then not a diagonalising rotation.  The Ritz vectors are unique up to a phase and
 * within degenerate eigenspaces. */
int tdh_subspace_diag(tdh_grid* g, int nst, const tdh_c128* psi_dev, const tdh_c128* hpsi_dev, tdh_c128* out_dev,
                      double* eig_host);

/* One Teter-preconditioned steepest-descent update of every state, independently (reading R19):
 *     eps_s = <psi|H psi>/<psi|psi>,  T_s = <psi|T psi>/<psi|psi>,  r = H psi - eps_s psi,
 *     p_hat(G) = K(t(G)/T_s) r_hat(G),  K(x) = (27+18x+12x^2+8x^3)/(27+18x+12x^2+8x^3+16x^4),  psi <- psi - lambda p
 * psi_dev: DEVICE block, updated in place; work_dev: DEVICE scratch block of the same size (holds the residuals
 * afterwards), must not overlap psi_dev; eig_host: HOST [nst], receives eps_s (before the update), or NULL.
 * One H application, one kinetic-only application and one preconditioner pass per state; no orthogonalisation
 * (tdh_orthonormalize).  Asynchronous unless eig_host is given. */
int tdh_sd_step(tdh_grid* g, int nst, tdh_c128* psi_dev, tdh_c128* work_dev, double lambda, double* eig_host);

/* Gradient along one axis, "a local operation in Fourier space":
 *     out = FFT^-1( i (G_a + k_a) FFT(psi) ),   axis a = 0, 1, 2   (frequency convention as in the kinetic term, no mask)
 * psi_dev, out_dev: DEVICE blocks of nst states, must not overlap.  Asynchronous on the handle's stream. */
int tdh_gradient(tdh_grid* g, int nst, const tdh_c128* psi_dev, int axis, tdh_c128* out_dev);

/* Eq. 11, per atom I of the projector table and axis a:
 *     F[I][a] = sum_s f_s ( <d_a psi_s | v_I | psi_s> + c.c. )
 * with v_I = the atom's Kleinman-Bylander projectors plus, if vloc_atoms_dev != NULL, its own local potential
 * vloc_atoms_dev[I][p] (DEVICE, natoms*n0*n1*n2 doubles).  occ_host: HOST [nst] or NULL (all 1).
 * forces_host: HOST [natoms][3].  This is +dE_I/dR_I of E_I = sum_s f_s <psi_s|v_I(r - R_I)|psi_s> at fixed orbitals
 * (reading R20).  One forward transform, three gradient chains and four projector gathers per state;
 * the non-local part is 2 Re of the projection coefficients of d_a psi against those of psi.  Synchronises. */
int tdh_forces(tdh_grid* g, int nst, const tdh_c128* psi_dev, const double* occ_host, const double* vloc_atoms_dev,
               double* forces_host);

/* ---- Slab decomposition of the grid over `world` ranks (Fig. 6: "the real-space is divided along the x
 * direction while the Fourier-space is split along" another one; "local transforms ... followed by a
 * redistribution of the data ... and the transform in the last dimension").  Rank r holds, of every state,
 *     real space:     planes x in [r n0/world, (r+1) n0/world), all y, z        block [nst][n0/world][n1][n2]
 *     Fourier space:  all k_x, the n1/world rows r n1/world .. of the WORK LAYOUT (the digit-permuted (k_y, k_z) order
 *                     the in-place transforms leave, see tdh_work_layout), all k_z            [nst][n0][n1/world][n2]
 * DESIGN.md section 14 says why the Fourier-space split is along y here (the paper draws z).  The redistribution is
 * not a separate copy: the kernel that produces a value stores it straight into the buffer of the rank that owns it
 * (device pointers of the peers: NVLink peer memory between GPUs, plain device memory when several ranks are emulated
 * on one device).  A Hamiltonian application of a rank is therefore four phases; the caller runs phase p on ALL ranks,
 * then a barrier across the ranks' streams, then phase p + 1:
 *     TDH_SLAB_PROJECT      partial Kleinman-Bylander projections over the rank's planes (nothing without projectors)
 *     TDH_SLAB_PLANES_FWD   sum of all ranks' partial projections (read from the peers, in rank order); forward (z,y)
 *                           transform of the rank's planes, every spectrum row stored to its owner
 *     TDH_SLAB_PENCILS      forward x, kinetic factor, inverse x on the rank's rows; every plane value stored to its owner
 *     TDH_SLAB_PLANES_INV   inverse (y,z) transform of the rank's planes, + V psi + V_nl psi, into hpsi
 * tdh_create_slab_grid: n, len, kpt, ecut, max_states, cuda_stream as tdh_create_grid (n is the FULL grid); world in
 * [2, 8] must divide n[0] and n[1]/2, and n[0]/world must be a multiple of the planes per tile (TDH_EUNSUPPORTED
 * otherwise).  On a slab handle tdh_set_potential takes the rank's planes of V ([n0/world][n1][n2]) and
 * tdh_set_projectors the sphere points inside the rank's planes with LOCAL flat indices ((x - x0) n1 + y) n2 + z and
 * the SAME atoms and channels on every rank (an atom may have no point on a rank); it frees and re-creates the rank's
 * partial-projection buffer, so it is a collective step: every rank stops using (and, with CUDA IPC, closes) the peers'
 * buffers first, and afterwards every rank calls tdh_slab_set_peers again -- until then the phase calls of this handle
 * return TDH_EINVAL; nst of a phase call is at most the
 * workspace chunk (max_states if that fits 4 GiB).  The other entry points that transform along x refuse slab handles. */
enum { TDH_SLAB_PROJECT = 0, TDH_SLAB_PLANES_FWD = 1, TDH_SLAB_PENCILS = 2, TDH_SLAB_PLANES_INV = 3 };
int tdh_create_slab_grid(const int n[3], const double len[3], const double kpt[3], double ecut, int max_states,
                         int rank, int world, void* cuda_stream, tdh_grid** out);
/* This rank's exchange buffers (DEVICE pointers owned by the handle): its Fourier-space slab, its real-space work
 * block, its partial-projection buffer (NULL until tdh_set_projectors; it changes with every tdh_set_projectors). */
int tdh_slab_buffers(tdh_grid* g, void** fs_dev, void** rs_dev, void** dpi_dev);
/* The same three buffers of ALL ranks, in rank order: HOST arrays of `world` DEVICE pointers valid on this device
 * (entry `rank` must be the handle's own).  dpi_dev may be NULL when no projectors are set.  Call after
 * tdh_set_projectors. */
int tdh_slab_set_peers(tdh_grid* g, void* const* fs_dev, void* const* rs_dev, void* const* dpi_dev);
/* One phase of hpsi = H psi on the rank's planes (psi_dev, hpsi_dev: DEVICE, nst*(n0/world)*n1*n2 complex128; hpsi_dev is
 * only used by TDH_SLAB_PLANES_INV).  Asynchronous on the handle's stream. */
int tdh_slab_apply_phase(tdh_grid* g, int phase, int nst, const tdh_c128* psi_dev, tdh_c128* hpsi_dev);
/* The distributed 3-D transform alone, two phases (barrier in between), in place on block_dev:
 *   sign -1: rank's planes [nst][n0/world][n1][n2] -> rank's spectrum rows [nst][n0][n1/world][n2] in work layout
 *   sign +1: the reverse, scaled by 1/(n0 n1 n2). */
int tdh_slab_fft_phase(tdh_grid* g, int sign, int phase, int nst, tdh_c128* block_dev);
/* CUDA IPC wrappers for one-process-per-GPU runs: export a handle-owned DEVICE buffer (tdh_slab_buffers) as a 64-byte
 * token, open a peer's token as a DEVICE pointer valid in this process (peer access is enabled lazily), close it. */
int tdh_ipc_export(void* dev_ptr, unsigned char handle[64]);
int tdh_ipc_import(const unsigned char handle[64], void** dev_ptr);
int tdh_ipc_close(void* dev_ptr);
/* The work layout: row rowmap[ky] / column colmap[kz] of a spectrum plane holds frequency index ky / kz
 * (HOST arrays of n1 and n2 ints). */
int tdh_work_layout(const tdh_grid* g, int* rowmap_host, int* colmap_host);

/* The same two operations with HOST buffers (pageable or pinned): the library stages state chunks through its own
 * pinned buffers, overlapping host<->device copies with the kernels, and returns when hpsi_host / psi_host is complete.
 * nst is not limited by max_states here (chunks are).  These are the end-to-end entry points timed by bench.py. */
int tdh_apply_hamiltonian_host(tdh_grid* g, int nst, const tdh_c128* psi_host, tdh_c128* hpsi_host);
int tdh_propagate_host(tdh_grid* g, int nst, tdh_c128* psi_host, double dt, int nsteps, int order);

/* Batched 3-D FFT alone (rows a1 / a3 of the scope table), in place on a DEVICE block.
 * sign = -1: forward, unnormalised, e^{-i G.r}; sign = +1: inverse, scaled by 1/(n0*n1*n2)   (reading R8). */
int tdh_fft3d(tdh_grid* g, int nst, tdh_c128* psi_dev, int sign);

/* Number of kernel launches the last tdh_apply_hamiltonian / tdh_propagate / *_host call of this handle enqueued. */
int tdh_last_launch_count(const tdh_grid* g);

/* Jacobi sweeps the last tdh_subspace_diag call of this handle needed. */
int tdh_last_jacobi_sweeps(const tdh_grid* g);

/* Seconds (device time, CUDA events on the handle's stream) spent in each kernel family during the last call, when
 * profiling was switched on with tdh_set_profiling(g, 1); profiling inserts events and synchronises at the end.
 * out[0..TDH_NKERNELS-1]; order given by tdh_kernel_name(i): nl_project, plane_fwd, xpencil, plane_inv, nl_scatter of the
 * tiled path, small_h = the one-launch on-chip kernel of 16^3 / 32^3 grids.  Off by default. */
#define TDH_NKERNELS 6
int tdh_set_profiling(tdh_grid* g, int on);
int tdh_last_kernel_seconds(const tdh_grid* g, double out[TDH_NKERNELS]);
const char* tdh_kernel_name(int i);

/* Allocate now what tdh_orthonormalize / tdh_subspace_diag (three n x n complex matrices for blocks of up to
 * rotation_states states; 0: none), tdh_sd_step (per-state reduction scratch), tdh_forces with per-atom local potentials
 * (forces_local_term != 0: three real grids) and the host entry points (host_buffers != 0: four staging buffers of at most
 * 512 MiB) would otherwise allocate at their first use, so that those calls allocate nothing either.
 * Synchronises the handle's stream when the rotation scratch grows.  TDH_EINVAL for rotation_states outside
 * [0, max_states], TDH_ENOMEM / TDH_ECUDA when an allocation fails (what was allocated before stays). */
int tdh_reserve(tdh_grid* g, int rotation_states, int forces_local_term, int host_buffers);

/* The overlap matrix of tdh_overlap for callers that may not allocate device memory and have no handle:
 *     S[i][j] = dV sum_p conj(a_i[p]) b_j[p],   i < na, j < nb,   row-major [na][nb] complex128
 * Meant for a host program whose own pool owns the device's memory (a cudaMalloc beside it fails or fragments it;
 * PAPER.md:326), for a time-stepping loop that cannot take cudaMalloc's device-wide synchronisation, and for anybody who
 * wants this one number check (are my states still orthonormal?) without creating a tdh_grid and its gigabytes of
 * workspace.  The call allocates nothing, on the host or on the device, and frees nothing: the split-K partial tiles live
 * in one fixed array of TDH_NOALLOC_SCRATCH_BYTES that is part of the library image, so every device that uses libtdh.so
 * gives up that much memory until the process exits.
 *   npts      number of grid points of a state (any value >= 1; no divisibility requirement)
 *   dv        the volume element dV (1.0 for a plain a^H b)
 *   na, nb    states in a and b, each in [1, TDH_NOALLOC_MAX_STATES]; larger blocks: TDH_EUNSUPPORTED, and the message says
 *             to use tdh_overlap
 *   a_dev, b_dev   DEVICE, na*npts / nb*npts complex128, on the CURRENT device (may be the same block: only the upper
 *                  tiles are then computed and mirrored)
 *   s_dev     DEVICE, na*nb complex128, must not overlap a or b
 *   cuda_stream    a cudaStream_t of the current device, or NULL
 * Asynchronous on that stream.  Slices of K are summed in order: the result is deterministic for given sizes on a given
 * GPU model, and equals tdh_overlap's up to the rounding of a different slice count.
 * SHARED SCRATCH: all calls of the process use the same array (it still holds the previous call's partial tiles; the
 * call overwrites every cell it reads, nothing has to be cleared).  Calls that can run at the same time on one device --
 * different streams, or different threads without ordering -- race on it; keep them on one stream or order them.
 * FIRST CALL: the first call on each device looks up the array's device address (and makes the runtime load the
 * library's kernels there); make it once at start-up with that device current, before any stream capture and before
 * the phase in which the program must not block. */
#define TDH_NOALLOC_MAX_STATES 256
#define TDH_NOALLOC_SCRATCH_BYTES (8u << 20)
int tdh_overlap_noalloc(size_t npts, double dv, int na, const tdh_c128* a_dev, int nb, const tdh_c128* b_dev,
                        tdh_c128* s_dev, void* cuda_stream);

/* Tuning knob: how many states are pushed through the kernel chain together (0 = library default: as many as the
 * handle's workspace of at most 4 GiB per buffer holds, a multiple of 8 when a block has to be split -- measured on
 * B200, longer launches are never slower than L2-resident small chunks). */
int tdh_set_chunk_states(tdh_grid* g, int chunk);

const char* tdh_last_error(void);                 /* thread-local, static storage; never NULL */

#ifdef __cplusplus
}
#endif
#endif /* TDH_H */

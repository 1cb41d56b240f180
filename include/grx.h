/* grx.h -- C ABI of the B200-native FP64 Valencia GRMHD right-hand side.
 *
 * The method is the right-hand-side evaluation of GRaM-X (arxiv 2210.17509; citations are PAPER.md
 * line numbers): "reconstruct -> Riemann -> flux divergence + source" (steps 2-4, l.127-132) of the
 * Valencia formulation, Eqs. (6)-(13) (l.86-114), with TVD/WENO5 reconstruction (l.130, l.134), the
 * HLLE solver (l.131, l.136) and an ideal-gas Gamma-law EOS (l.138).  Readings of everything the paper
 * leaves open (R1..R32) are listed in DESIGN.md.
 *
 * Conventions shared by every entry point
 * ---------------------------------------
 *  - Every array pointer is a DEVICE pointer to FP64 unless it says HOST.  The caller owns all memory;
 *    the library never allocates, frees or keeps user memory.  grx_valencia_rhs and grx_prim2con need no
 *    workspace; the host, time-stepping and constrained-transport entry points take one from the caller.
 *  - State: none between calls, except three debug/plumbing items that are stated where they are declared: the
 *    process-wide kernel selector (grx_set_variant, default AUTO), the per-thread fallback counter pointer
 *    (grx_debug_set_fallback_counter) and two per-thread CUDA streams that grx_valencia_rhs_host creates on
 *    first use; plus the fixed device array of grx_valencia_rhs_ct_static and its per-device address.  No environment
 *    variable is read.  Entry points may be called from several host threads and on
 *    several devices (the current device of the calling thread is used).
 *  - Layout: structure of arrays, x fastest, ghost zones included, boxes contiguous:
 *        a[box][field][k][j][i],   i in [0,Nx), j in [0,Ny), k in [0,Nz),   N* = n* + 2*nghost,
 *    interior cell (i,j,k) of the paper's block (l.184) sits at (i+nghost, j+nghost, k+nghost).
 *  - Fields (fixed order):
 *        prim  [8] : rho, v^x, v^y, v^z, eps, B^x, B^y, B^z     (P of l.118; Valencia v^i, Eq. 10 l.98;
 *                                                               eps = specific internal energy, R1)
 *        metric[10]: alp, beta^x, beta^y, beta^z, g_xx, g_xy, g_xz, g_yy, g_yz, g_zz   (ADM, l.56)
 *        K     [6] : K_xx, K_xy, K_xz, K_yy, K_yz, K_zz   (d_t g_ij = -2 alp K_ij + Lie_beta g_ij, R12)
 *        cons/out[8]: D, S_x, S_y, S_z, tau, calB^x, calB^y, calB^z  (densitised, Eqs. 6-9 l.88-94)
 *    Metric and K are co-located with the fluid at cell centres (R6), except in the two vertex-centred entry points
 *    (grx_valencia_rhs_vertex, grx_tmunu_vertices: R31 / R32), which say so.
 *  - Calls are asynchronous on `cuda_stream` (a cudaStream_t; NULL = the legacy default stream); results
 *    are valid after that stream is synchronised.
 *  - Errors: every entry point returns a code, never aborts or throws.  Arguments are validated on the
 *    host BEFORE any launch (nothing is written on GRX_ERR_INVALID_ARG).  CUDA launch failures map to
 *    GRX_ERR_CUDA.  Inputs are not checked for physical admissibility on the device: an unphysical
 *    cell-centre state gives NaN/Inf there, exactly as the equations do.
 *  - There is NO CPU fallback: without a CUDA device every compute entry point returns GRX_ERR_CUDA.
 */
#ifndef GRX_H
#define GRX_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    int nx, ny, nz; /* interior cells per box, each >= 1                    */
    int nbox;       /* boxes in this call, >= 1, stored back to back         */
} grx_grid;

enum { GRX_RECON_MINMOD = 0, GRX_RECON_MC = 1, GRX_RECON_WENO5 = 2 };
enum { GRX_OK = 0, GRX_ERR_INVALID_ARG = 1, GRX_ERR_CUDA = 2, GRX_ERR_UNSUPPORTED = 3 };

/* Kernel selector (grx_set_variant), a debugging and measurement aid.
 *   AUTO    the product path: the TMA kernel (csrc/grx_tma.cu: planes staged in shared memory by cp.async.bulk.tensor,
 *           shared-memory z rings) when the arrays qualify -- Nx = nx + 2 nghost even and prim, metric, K 16-byte
 *           aligned, as TMA needs 16-byte global strides -- and the LDG kernel otherwise;
 *   SIMPLE  cross-check traversal: one thread per cell, every thread evaluates its own six faces;
 *   LDG     always the round-1 kernel (csrc/grx_fused.cu: same decomposition, operands through L1 with __ldg);
 *   TMA     always the TMA kernel; grx_valencia_rhs returns GRX_ERR_UNSUPPORTED when the arrays do not qualify. */
enum { GRX_VARIANT_AUTO = 0, GRX_VARIANT_SIMPLE = 1, GRX_VARIANT_LDG = 2, GRX_VARIANT_TMA = 3 };

/* d/dt of the conserved variables on the interior cells of every box.
 *
 * Computes, per direction d = x,y,z:
 *   face metric = 1/2 (cell- + cell+) (l.130, R6/R7); reconstruction of the 8 primitives to both sides of
 *   every face with `recon` (minmod/MC: l.134, l.255; WENO5 Jiang-Shu: l.134, ref [32]); first-order
 *   fallback of an inadmissible side (R5); conserved state Eqs. (6)-(10) and flux Eq. (12) per side
 *   (l.88-108); fast-magnetosonic speeds (R8); HLLE flux (l.131, R9); out -= (F_{f+1} - F_f)/dx_d;
 * then adds the geometric sources of Eq. (13) (l.112) in 3+1 form (R12-R14) with 4th-order centred
 * metric derivatives, evaluated from the cell-centre primitives.
 *
 *   grid    HOST pointer.
 *   prim    [nbox][8 ][Nz][Ny][Nx]  in.   Ghosts must be filled by the caller (l.170, l.222).
 *   metric  [nbox][10][Nz][Ny][Nx]  in.
 *   K       [nbox][6 ][Nz][Ny][Nx]  in.
 *   dx      HOST pointer to 3 cell sizes, each > 0 (R11).
 *   nghost  ghost width on every side: >= 3 for WENO5, >= 2 for minmod/MC (R29).
 *   recon   GRX_RECON_*.
 *   gamma   Gamma-law index, > 1 (l.138).
 *   out     [nbox][8][Nz][Ny][Nx]   out.  Interior cells are overwritten; ghost cells are not touched
 *           (R23).  Must not alias an input.
 * Returns GRX_OK, GRX_ERR_INVALID_ARG (null pointer, n < 1, nbox < 1, nghost too small, unknown recon,
 * gamma <= 1, dx <= 0, a box larger than 2^31-1 cells), GRX_ERR_UNSUPPORTED (only with GRX_VARIANT_TMA forced on
 * arrays that do not qualify) or GRX_ERR_CUDA. */
int grx_valencia_rhs(const grx_grid* grid, const double* prim, const double* metric, const double* K,
                     const double dx[3], int nghost, int recon, double gamma, double* out, void* cuda_stream);

/* Same computation for HOST arrays (end-to-end entry point): copies prim, metric and K to the device
 * workspace, evaluates the right-hand side there and copies the result back.  Blocks with more than 32 planes
 * along z are processed as a pipeline of 32-plane slabs: the upload of the next slab, the kernel of the current
 * one and the download of the previous one overlap on three streams (two internal ones per host thread and
 * device, created on first use and kept, ordered after / before `cuda_stream` by events); the results are bitwise
 * those of the device entry point on the interior cells.  Ghost cells of `out_host` (unlike those of the device entry
 * point's `out`) are NOT preserved: in the pipelined case the planes k = nghost .. nz + nghost - 1 are copied back whole, so
 * their x and y ghost cells receive whatever the workspace held, and the z ghost planes are left alone; for blocks of <= 32
 * planes, or while a debug fallback counter is set, the whole array is copied back.  The host arrays have the layout above
 * and should be page-locked for the copies to be asynchronous.
 *   workspace        DEVICE pointer, at least grx_host_workspace_bytes(grid, nghost) bytes, owned by the caller.
 * Results are valid in out_host after `cuda_stream` is synchronised. */
size_t grx_host_workspace_bytes(const grx_grid* grid, int nghost);
int grx_valencia_rhs_host(const grx_grid* grid, const double* prim_host, const double* metric_host,
                          const double* K_host, const double dx[3], int nghost, int recon, double gamma,
                          double* out_host, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Conserved variables from the primitives, Eqs. (6)-(9), with the CELL-CENTRE metric,
 * on ALL cells including ghosts (step 2 of the initialisation, l.120-123).
 *   cons    [nbox][8][Nz][Ny][Nx]   out.  nghost >= 0. */
int grx_prim2con(const grx_grid* grid, const double* prim, const double* metric, int nghost, double gamma,
                 double* cons, void* cuda_stream);

/* SUPPORT CODE for short evolutions (R21/R22; not on the graded path): primitives from conserved
 * variables for the Gamma-law EOS by a bracketed Newton solve in z = rho h W^2 (stand-in for the paper's
 * 3D-NR scheme, l.142-146), on ALL cells including ghosts.
 *   prim    [nbox][8][Nz][Ny][Nx]   out.
 *   nfail   DEVICE pointer to one unsigned long long, or NULL: incremented (atomically) by the number of
 *           cells whose solve did not converge; the caller zeroes it. */
int grx_con2prim(const grx_grid* grid, const double* cons, const double* metric, int nghost, double gamma,
                 double* prim, unsigned long long* nfail, void* cuda_stream);

/* SUPPORT CODE: y[interior] = a*x[interior] + b*(y[interior] + dt*rhs[interior]) on 8-field arrays --
 * the building block of the SSP-RK2 stages (l.125, R21).  x may equal y. */
int grx_rk_axpy(const grx_grid* grid, int nghost, double a, const double* x, double b, double dt,
                const double* rhs, double* y, void* cuda_stream);

/* NEXT-1: `nsteps` time steps of the method of lines around the right-hand
 * side, entirely on the device and on the caller's stream -- no host round trip between stages.  Every stage is
 *   L = grx_valencia_rhs(prim);   U <- a U0 + b (U + h L) on the interior, FUSED with con2prim of the new U (step 1 of the
 *   paper's RHS evaluation, l.129; Gamma-law, R22) and, for RK4, with the accumulation of U0 + dt/6 (k1 + 2k2 + 2k3 + k4);
 *   ghost fill of the 8 primitives at the outer boundary (l.170): GRX_BC_COPY (von Neumann "copy", l.255) or
 *   GRX_BC_PERIODIC (l.329).
 * rk_order 2 = SSP-RK2 / Heun (R21), 4 = classical RK4 (l.255, l.335).
 *   cons    [nbox][8][Nz][Ny][Nx]  in/out: conserved variables on the INTERIOR cells (e.g. from grx_prim2con); ghosts unused.
 *   prim    [nbox][8][Nz][Ny][Nx]  in/out: primitives with FILLED ghosts, consistent with cons; on return those of the new
 *           time level, ghosts filled.
 *   metric, K, dx, nghost, recon, gamma: as for grx_valencia_rhs (static spacetime: they are not evolved).
 *   workspace  DEVICE pointer, at least grx_step_workspace_bytes(grid, nghost, rk_order) bytes (2 arrays of the size of
 *           cons for RK2, 3 for RK4), owned by the caller.
 *   nfail   DEVICE pointer to one unsigned long long (caller-zeroed) or NULL: incremented by the number of cells whose
 *           con2prim did not converge.
 * Returns GRX_OK, GRX_ERR_INVALID_ARG or GRX_ERR_CUDA. */
enum { GRX_BC_COPY = 0, GRX_BC_PERIODIC = 1 };
size_t grx_step_workspace_bytes(const grx_grid* grid, int nghost, int rk_order);
int grx_step_rk(const grx_grid* grid, double* cons, double* prim, const double* metric, const double* K,
                const double dx[3], int nghost, int recon, double gamma, double dt, int rk_order, int bc, int nsteps,
                void* workspace, size_t workspace_bytes, unsigned long long* nfail, void* cuda_stream);

/* NEXT-2: the right-hand side with constrained transport for the magnetic field (PAPER.md l.287,
 * l.299, l.315; face / edge locations l.194-196).  The paper prints no algorithm; reading R30 is flux-CT of the
 * cell-centred calB^i: with F^j(calB^i) = eps_ijk E_k, the EMF on a cell edge is the mean of the four HLLE face fluxes that
 * touch it, the flux through a face is replaced by the mean of the two edge EMFs on it, and out[5..7] = d calB^i/dt becomes
 * the difference of the replaced fluxes (the vertex-centred divergence of the update vanishes to rounding).  out[0..4] are
 * those of grx_valencia_rhs, bit for bit.  The face fluxes come out of the same kernel launch as the right-hand side (TMA
 * kernel) plus a kernel for the one layer of grid lines next to the block, whose faces the edge averages reach: prim and
 * metric must be filled on the ghost cells as for grx_valencia_rhs, no wider.
 *   workspace  DEVICE pointer, at least grx_ct_workspace_bytes(grid, nghost) bytes (six face-flux arrays), owned by the
 *              caller; holds F^x(B^y), F^x(B^z), F^y(B^x), F^y(B^z), F^z(B^x), F^z(B^y) at the low face of each cell on return.
 * Other arguments, return codes and asynchrony as for grx_valencia_rhs. */
size_t grx_ct_workspace_bytes(const grx_grid* grid, int nghost);
int grx_valencia_rhs_ct(const grx_grid* grid, const double* prim, const double* metric, const double* K,
                        const double dx[3], int nghost, int recon, double gamma, double* out, void* workspace,
                        size_t workspace_bytes, void* cuda_stream);

/* grx_valencia_rhs_ct for callers that have no device memory to give and may not ask the driver for any.
 *
 * Who that is: in the setting this method comes from, one component of the host code owns device memory -- the paper's
 * driver "handles all data movement and memory allocations" (l.154) and calls user functions on blocks of data -- and such
 * drivers commonly reserve most of HBM for their own arena at start-up, so cudaMalloc may have nothing left to return.  A
 * routine called from inside that time loop, through an interface that passes field pointers only, or from a region where
 * the device-wide synchronisation implied by cudaMalloc / cudaFree would stall every other stream, cannot size and
 * allocate the six face-flux arrays that grx_valencia_rhs_ct wants as `workspace`.  This entry point keeps those arrays inside the library instead:
 * in ONE fixed array of GRX_CT_STATIC_MAX_BYTES (16 MiB) of device memory that is part of the loaded library image.  Every
 * GPU on which the process uses the library holds these 16 MiB from the moment the library's code is loaded there until
 * the process exits, whether or not this entry point is ever called.
 *
 *   - It calls no cudaMalloc, cudaFree or any other allocating routine, on any call.  prim, metric, K and out are the
 *     caller's, exactly as for grx_valencia_rhs_ct; results are the same bits as grx_valencia_rhs_ct gives.
 *   - Limit: 6 * (nx + 2 nghost)(ny + 2 nghost)(nz + 2 nghost) * nbox * 8 bytes <= GRX_CT_STATIC_MAX_BYTES, i.e. at most
 *     349 525 cells (ghosts included) summed over the boxes of the call -- one 64^3 block with 3 ghost cells (70^3 = 343 000)
 *     fits, so do 4 x 38^3.  A larger call returns GRX_ERR_INVALID_ARG ("... exceeds the static scratch ...") and launches
 *     nothing: split it into several calls, or use grx_valencia_rhs_ct with your own workspace.
 *   - First call on each device: the library looks up the device address of the array once per device (with the calling
 *     thread's current device) and keeps it.  That look-up makes the CUDA runtime load the library's device code on that
 *     device if it has not yet done so.  Make this first call during start-up, before any stream capture begins.
 *   - All calls on one device share the one array, from every thread and every stream.  Two calls whose kernels can be on
 *     the GPU at the same time (different streams without an ordering between them, or two host threads) overwrite each
 *     other's face fluxes and both results are garbage: order them on one stream or with events.  Calls on different
 *     devices do not interact.
 *   - The array keeps what the previous call left in it.  Nothing in it has to start at zero: each call writes every
 *     face flux it later reads (faces of the interior grid lines by the right-hand-side kernel, the one layer next to the
 *     block by the face kernel) before the curl kernel runs, so stale contents are never read.  The face fluxes are not
 *     returned; a caller that wants them uses grx_valencia_rhs_ct.
 * grx_ct_static_max_bytes() returns GRX_CT_STATIC_MAX_BYTES (for bindings that cannot see the macro).
 * Other arguments, return codes and asynchrony as for grx_valencia_rhs_ct. */
#define GRX_CT_STATIC_MAX_BYTES ((size_t)16 << 20)
size_t grx_ct_static_max_bytes(void);
int grx_valencia_rhs_ct_static(const grx_grid* grid, const double* prim, const double* metric, const double* K,
                               const double dx[3], int nghost, int recon, double gamma, double* out, void* cuda_stream);

/* NEXT-4 (PAPER.md l.222-230 ghost-zone fill between blocks, l.371 "start the computations of those
 * cells ... which do not need ghost cells while ghost cells ... are getting filled, and then compute the remaining cells
 * thereafter"): the pieces a slab decomposition along z needs to overlap the ghost exchange with the interior update.
 * paper_2210_17509_b200/halo.py composes them with torch.distributed point-to-point transfers.
 *
 * grx_valencia_rhs_zrange: the right-hand side on the interior planes k_begin <= k < k_end only (nbox = 1); every plane gets
 *   the bits of the whole-block call (same kernel choice, same arithmetic per cell).  Planes g <= k < nz - g read no z ghost
 *   plane and can run while those are in flight; [0, g) and [nz - g, nz) follow when they have arrived.
 * grx_halo_z: pack (unpack = 0) the nghost lowest (side 0) or highest (side 1) INTERIOR planes of the 8 primitive fields into
 *   buf[nbox][8][nghost][Ny][Nx], or unpack (unpack = 1) buf into the low (side 0) / high (side 1) z GHOST planes.  Planes
 *   travel with their x and y ghost cells (fill those first).  buf: DEVICE, grx_halo_z_bytes(grid, nghost) bytes; nbox <= 8191.
 * grx_fill_ghosts: the ghost fill of grx_step_rk as a call of its own; dirs = mask of the directions filled here (bit 0 = x,
 *   1 = y, 2 = z): a z-slab rank fills x and y (dirs = 3) and receives z.
 * grx_rk_stage: the stage update of grx_step_rk as a call of its own: Uout = a Ua + b (Ub + h L) on the interior cells,
 *   acc += wdt L if acc is non-NULL, prim = con2prim(Uout) (Gamma-law, R22); nfail as for grx_con2prim. */
int grx_valencia_rhs_zrange(const grx_grid* grid, const double* prim, const double* metric, const double* K,
                            const double dx[3], int nghost, int recon, double gamma, double* out, int k_begin, int k_end,
                            void* cuda_stream);
size_t grx_halo_z_bytes(const grx_grid* grid, int nghost);
int grx_halo_z(const grx_grid* grid, double* prim, int nghost, int side, int unpack, double* buf, void* cuda_stream);
/* grx_halo_z_pull: the peer-memory transport of the same exchange: one kernel that fills both sets of z ghost planes of `prim`
 * by reading the neighbours' arrays directly -- below / above: DEVICE pointers to the prim arrays (same grid, same layout) of
 * the slabs below and above, on this device or on a peer device whose memory is accessible from this one (NVLink peer
 * access enabled by the caller).  No pack buffer and no staging copy.  The neighbours' x / y ghosts must be filled and their
 * interior planes final when the kernel runs (order it with events).  A slab that is its own neighbour passes prim itself. */
int grx_halo_z_pull(const grx_grid* grid, double* prim, int nghost, const double* below, const double* above, void* cuda_stream);
int grx_fill_ghosts(const grx_grid* grid, double* prim, int nghost, int bc, int dirs, void* cuda_stream);
int grx_rk_stage(const grx_grid* grid, int nghost, double a, const double* Ua, double b, const double* Ub, double h,
                 const double* L, double* Uout, double* acc, double wdt, const double* metric, double gamma, double* prim,
                 unsigned long long* nfail, void* cuda_stream);

/* NEXT-3: the paper's own centring of the spacetime fields -- "stored on vertices",
 * "known at the cell vertices and ... interpolated linearly to the face centers" (l.130); T^{mu nu} "stored as samples at the
 * cell vertices" from fluid variables brought there by "a 4th-order symmetric 3D interpolation" (l.84, l.323).  Readings R31 /
 * R32.  Vertex arrays: metric_v[nbox][10][Nz+1][Ny+1][Nx+1], K_v[nbox][6][Nz+1][Ny+1][Nx+1], vertex (I, J, K) = the
 * low corner of cell (I, J, K) (indices with ghosts).
 *
 * grx_valencia_rhs_vertex: grx_valencia_rhs with face metric = mean of the 4 vertices of the face, cell-centre metric and K_ij
 *   = mean of the 8 vertices of the cell, metric derivatives = [27 (m(+1/2) - m(-1/2)) - (m(+3/2) - m(-3/2))] / (24 dx) of the
 *   transverse 4-vertex means.  prim, dx, nghost, recon, gamma, out, errors: as for grx_valencia_rhs.  Runs on the tile
 *   traversal of the LDG kernel with vertex loads (GRX_VARIANT_SIMPLE: one thread per cell, the cross-check).
 * grx_tmunu_vertices: T[nbox][10][Nz+1][Ny+1][Nx+1] = T^{00}, T^{0x}, T^{0y}, T^{0z}, T^{xx}, T^{xy}, T^{xz}, T^{yy}, T^{yz}, T^{zz}
 *   (Eq. 5, l.80) at the (n+1)^3 vertices of the interior cells of every box; other entries are not written.  The 8
 *   primitives are interpolated to the vertex with the tensor product of (-1, 9, 9, -1)/16 over the 4 x 4 x 4 cells around it
 *   (nghost >= 2), the metric is the vertex's own sample. */
int grx_valencia_rhs_vertex(const grx_grid* grid, const double* prim, const double* metric_v, const double* K_v,
                            const double dx[3], int nghost, int recon, double gamma, double* out, void* cuda_stream);
int grx_tmunu_vertices(const grx_grid* grid, const double* prim, const double* metric_v, int nghost, double gamma, double* T,
                       void* cuda_stream);

/* grx_step_rk with constrained transport (NEXT-1 + NEXT-2; the paper's multi-dimensional tests, l.287, l.299): every right-hand
 * side of every stage is grx_valencia_rhs_ct, so the vertex-centred divergence of calB stays what it was initially, to
 * rounding.  Arguments as for grx_step_rk; workspace: at least grx_step_ct_workspace_bytes(grid, nghost, rk_order) bytes (the
 * arrays of grx_step_rk followed by the six face-flux arrays). */
size_t grx_step_ct_workspace_bytes(const grx_grid* grid, int nghost, int rk_order);
int grx_step_rk_ct(const grx_grid* grid, double* cons, double* prim, const double* metric, const double* K,
                   const double dx[3], int nghost, int recon, double gamma, double dt, int rk_order, int bc, int nsteps,
                   void* workspace, size_t workspace_bytes, unsigned long long* nfail, void* cuda_stream);

/* Debug: if `counter` (DEVICE pointer to one unsigned long long, caller-zeroed) is non-NULL, later
 * grx_valencia_rhs calls of this host thread add to it the number of face sides that took the R5
 * first-order fallback.  NULL switches counting off (the default; counting costs a few atomics). */
int grx_debug_set_fallback_counter(unsigned long long* counter);

/* Debug (the call SURVEY.md section 8(b) sketches for the R5 count): copies the counter registered by this host thread
 * with grx_debug_set_fallback_counter to *host_out (HOST pointer), ordered after the work already enqueued on `cuda_stream`,
 * and synchronises that stream.  The value is what has accumulated since the caller last zeroed the counter: zero it
 * before the call whose fallbacks are wanted to get "the count of the last call".  GRX_ERR_INVALID_ARG if host_out is NULL
 * or no counter is registered on this thread; GRX_ERR_CUDA if the copy fails. */
int grx_debug_fallback_count(unsigned long long* host_out, void* cuda_stream);

/* Selects the kernel used by later grx_valencia_rhs calls of this PROCESS (default GRX_VARIANT_AUTO). */
int grx_set_variant(int variant);

/* Accuracy self-test of the division-free reciprocal / rsqrt / sqrt helpers the kernels use:
 * y[0..n) = 1/x, y[n..2n) = 1/sqrt(x), y[2n..3n) = sqrt(x) for x[0..n) > 0 (DEVICE pointers). */
int grx_selftest_math(const double* x, double* y, size_t n, void* cuda_stream);

/* Thread-local description of the last non-OK return of this thread ("" if none). */
const char* grx_last_error(void);

/* Library version: major*10000 + minor*100 + patch. */
int grx_version(void);

/* Compile-time conventions (R4, R5), exported so tests can assert that both implementations agree. */
double grx_weno_eps(void);
double grx_v2max(void);

#ifdef __cplusplus
}
#endif
#endif /* GRX_H */

/*
 * acm.h -- C ABI of libacm: the per-time-step coupled lattice-Boltzmann update of the
 * conservative Allen-Cahn model (ACM) for immiscible fluids at high density ratio,
 * arXiv 2012.06144 (PAPER.md "P:<line>"), as hand-written CUDA kernels for sm_100a (B200).
 *
 * What one time step computes (Algorithm 2; equations of section 3):
 *   1. phase-field LB step: stream-pull the populations h_i, phi = sum_i h_i (eq. 7),
 *      isotropic finite-difference grad phi (eq. 23), interface normal n, Allen-Cahn forcing
 *      (eq. 5), MRT collision (eq. 4), store h and phi               -- ONE kernel;
 *   2. hydrodynamic LB step: velocity-based populations g_i, rho(phi) (eq. 8),
 *      chemical potential (eq. 17), surface-tension, pressure, viscous and body force
 *      (eqs. 13-18, 30), tau(phi) (eqs. 20-21), velocity (eq. 22), MRT collision
 *      (eqs. 10-12, 25), streaming, store g and u                          -- ONE kernel.
 * Readings of the paper where it is silent or garbled are listed in DESIGN.md.
 *
 * Conventions
 *   - All field arrays are structure-of-arrays with x fastest: element (q, x, y, z) of a
 *     population array lives at ((q*nz + z)*ny + y)*nx + x; u is component-major (3 planes).
 *   - Element type of every `void*` field pointer follows `precision` of acm_create
 *     (ACM_F64: double, ACM_F32: float).
 *   - Direction order ("canonical order") of the population arrays exchanged through
 *     acm_get_pdfs: rest; (+x,-x,+y,-y,+z,-z); the 12 edge directions
 *     (+1,+1,0)(-1,-1,0)(+1,-1,0)(-1,+1,0)(+1,0,+1)(-1,0,-1)(+1,0,-1)(-1,0,+1)
 *     (0,+1,+1)(0,-1,-1)(0,+1,-1)(0,-1,+1); the 8 corner directions
 *     (+1,+1,+1)(-1,-1,-1)(+1,+1,-1)(-1,-1,+1)(+1,-1,+1)(-1,+1,-1)(-1,+1,+1)(+1,-1,-1).
 *     D3Q15 = rest+axis+corner, D3Q19 = rest+axis+edge, D3Q27 = all.
 *     D2Q9 (the two-dimensional instance the paper measures in Fig. 5) = rest, (+x,-x,+y,-y),
 *     (+1,+1)(-1,-1)(+1,-1)(-1,+1); it is used for BOTH LB steps on a grid with nz = 1 and gravity[2] = 0;
 *     u keeps three components, the third stays 0.
 *   - Ownership: the CALLER owns all device memory.  The library never allocates device
 *     memory; acm_create carves the caller's workspace.  The context (host memory) is
 *     freed by acm_destroy only.
 *   - Pointers marked [device] must be device pointers valid on the current CUDA device,
 *     pointers marked [host] are ordinary host pointers (pinned memory makes the copies
 *     asynchronous but is not required).
 *   - Every call returns an ACM_* code and never throws; acm_last_error() describes the
 *     last failure of the calling thread.  CUDA errors are sticky: once a launch failed,
 *     every later call on the context returns ACM_ECUDA.
 *   - All work is issued on the stream given to acm_create; calls are asynchronous with
 *     respect to the host unless stated otherwise.
 */
#ifndef ACM_H_
#define ACM_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct acm_ctx acm_ctx; /* opaque; owns no device memory */

enum { ACM_OK = 0, ACM_EINVAL = 1, ACM_ESTATE = 2, ACM_ECUDA = 3, ACM_EUNSTABLE = 4 };
enum { ACM_D2Q9 = 9, ACM_D3Q15 = 15, ACM_D3Q19 = 19, ACM_D3Q27 = 27 };
/* set: half-way bounce-back no-slip walls on both faces of that axis; clear: periodic */
enum { ACM_WALL_X = 1, ACM_WALL_Y = 2, ACM_WALL_Z = 4 };
enum { ACM_F64 = 0, ACM_F32 = 1 };

/* Bytes of device workspace acm_create needs for this configuration (two grids of h and g,
 * two phi buffers, u, a 5N staging area for the *_host calls and reduction scratch), or 0 if
 * the configuration is invalid. */
size_t acm_workspace_bytes(int nx, int ny, int nz, int stencil_phase, int stencil_hydro, int precision);

/* Creates a context.  Parameters follow the paper's statement of the problem:
 *   nx,ny,nz        grid size in cells (each >= 1; nx*ny*nz < 2^31)
 *   stencil_phase   lattice of h: ACM_D3Q15 | ACM_D3Q19 | ACM_D3Q27, or ACM_D2Q9 for both
 *   stencil_hydro   lattice of g: ACM_D3Q19 | ACM_D3Q27 (ACM_D3Q15 also accepted)
 *   rho_H, rho_L    densities of the heavy / light phase, rho_H >= rho_L > 0   (eq. 8)
 *   sigma           surface tension >= 0; beta = 12 sigma/xi, kappa = 3 sigma xi/2
 *   xi              interface thickness > 0
 *   M               mobility > 0; tau_phi = M/c_s^2 (eq. 2), first-order moments of h relax
 *                   with 1/(tau_phi + 1/2)
 *   nu_H, nu_L      kinematic viscosities > 0; tau = nu/c_s^2 (eq. 19) interpolated linearly
 *                   in phi (eq. 20), s_nu = 1/(tau + 1/2) (eq. 21)
 *   gravity[3]      [host] acceleration g of the body force F_b = rho g (eq. 30); NULL = 0
 *   wall_flags      OR of ACM_WALL_*
 *   precision       ACM_F64 (the paper's precision) or ACM_F32
 *   workspace       [device] >= acm_workspace_bytes() bytes, 256-byte aligned, caller-owned,
 *                   must outlive the context
 *   cuda_stream     a cudaStream_t (NULL = legacy default stream)
 * Errors: ACM_EINVAL for any violated constraint above (and *out = NULL). */
int acm_create(acm_ctx** out, int nx, int ny, int nz, int stencil_phase, int stencil_hydro,
               double rho_H, double rho_L, double sigma, double xi, double M, double nu_H, double nu_L,
               const double gravity[3], unsigned wall_flags, int precision,
               void* workspace, void* cuda_stream);

/* Options of acm_create_opt / acm_workspace_bytes_opt (OR of):
 *   ACM_OPT_INPLACE   one grid per population set instead of two (P:258 uses two): the streaming
 *                     of h and g follows the in-place AA pattern the paper names as the open
 *                     alternative; phi stays double-buffered because its finite-difference
 *                     stencil is non-local.  Same results, same bytes moved per step, half the
 *                     population memory.
 *   ACM_OPT_PHASE_SRT single-relaxation-time phase-field collision, Omega^h = omega_phi I: the set-up of
 *                     the paper's benchmarks ("D3Q15 SRT LB scheme for the interface tracking",
 *                     P:285) instead of the MRT operator of section 3.1.
 *   ACM_OPT_UNFUSED   Algorithm 1 of the paper, kept as a measured comparison for the fusion
 *                     claim of section 5: the time step as six kernels (stream h, update
 *                     phi, collide h, stream g, update u, collide g) instead of two.  Same results as
 *                     the default (Algorithm 2); every population array is read three times and
 *                     written twice per step.  Needs 3N more workspace (u is double-buffered); cannot
 *                     be combined with ACM_OPT_INPLACE (ACM_EINVAL).
 *   ACM_OPT_BULK_ONE  the other reading of "we relax the second order moments with s_nu ... all other moments are
 *                     relaxed by one" (A4/A26): only the five deviatoric second-order
 *                     moments relax with s_nu, their trace (the bulk moment) with 1.  Same shear viscosity,
 *                     bulk viscosity 1/9 instead of 2 nu/3.  Not with ACM_OPT_UNFUSED or slabs (ACM_EINVAL).
 *   ACM_OPT_MOMENTS   moment representation of the state (beyond the paper, last paragraph).  The paper's
 *                     collisions relax every moment of h beyond the first order and of g beyond the second order
 *                     with rate 1, so the post-collision populations of a cell are
 *                     w_i [A + e_i.b + e_i e_i : T] with 4 (h: A, b; T = 4.5 phi u u^T follows from phi and u) and
 *                     10 (g: A, b, T) numbers.  The workspace then holds those instead of Q_h + Q_g populations and the
 *                     pull of the next step rebuilds the one population each neighbour contributes; u is
 *                     double-buffered.  Same time step, same results up to rounding (same bars against the oracle);
 *                     128 + 216 B of traffic per cell and step for every lattice instead of 8 (2 Q_h + 5) +
 *                     8 (2 Q_g + 7).  ACM_F64 only; not with ACM_OPT_INPLACE / ACM_OPT_UNFUSED / ACM_OPT_PHASE_SRT
 *                     (SRT keeps every moment) or slabs (ACM_EINVAL); acm_set_pdfs returns ACM_EINVAL (arbitrary
 *                     populations have no such representation), acm_get_pdfs rebuilds the populations. */
enum { ACM_OPT_INPLACE = 1, ACM_OPT_PHASE_SRT = 2, ACM_OPT_UNFUSED = 4, ACM_OPT_BULK_ONE = 8, ACM_OPT_MOMENTS = 16, ACM_OPT_ALL = 31 };
size_t acm_workspace_bytes_opt(int nx, int ny, int nz, int stencil_phase, int stencil_hydro, int precision,
                               unsigned options);
/* acm_create with options; acm_create(...) == acm_create_opt(..., options = 0, ...). */
int acm_create_opt(acm_ctx** out, int nx, int ny, int nz, int stencil_phase, int stencil_hydro,
                   double rho_H, double rho_L, double sigma, double xi, double M, double nu_H, double nu_L,
                   const double gravity[3], unsigned wall_flags, int precision, unsigned options,
                   void* workspace, void* cuda_stream);

/* Equilibrium initialiser ("Initialisation of all fields", Alg. 2 line 1):
 * phi-field <- phi, u-field <- u, h_i <- phi Gamma_i(u) (eq. 6), g_i <- Gamma_i(u) - w_i
 * (eq. 12 with p* = 0).  phi: [device] N values; u: [device] 3N values, component-major.
 * Asynchronous, with one exception: for ACM_F32 with the automatic reference phase (acm_set_reference_phase = -1, the
 * default, on a context that is not a slab) the call reduces mean(phi) on the device and SYNCHRONISES the stream to
 * read it before it launches the initialiser. */
int acm_init(acm_ctx*, const void* phi, const void* u);

/* Velocity of eq. 22 by `sweeps` >= 1 sweeps of the fixed point u <- sum_i g_i e_i + F(u)/(2 rho): eq. 22 is implicit
 * because the viscous force (eq. 18) contains g^eq(u).  sweeps = 1 (default, A10): F_mu is
 * evaluated once with the velocity of the previous time step; sweeps = k re-evaluates it k-1 times with the velocity
 * just obtained (A27).  Takes effect from the next step.  ACM_EINVAL for sweeps outside 1..64, or > 1 on a
 * slab / with ACM_OPT_UNFUSED. */
int acm_set_subiter(acm_ctx*, int sweeps);

/* ACM_OPT_MOMENTS only (ACM_ESTATE otherwise): which kernels advance the moment representation.
 *   mode  -1 (default) automatic: the tiled kernels for three-dimensional grids of at least 2^21 cells, else the
 *            direct ones; 0 = direct kernels (one thread per cell, the coefficients of the neighbours gathered through
 *            L1/L2); 1 = tiled kernels: a block owns a 32 x 8 tile of columns and marches along z with a window of planes
 *            in shared memory -- the phase-field kernel (and the D3Q27 hydrodynamic kernel) gathers from coefficient
 *            planes staged by cp.async, the D3Q15 / D3Q19 hydrodynamic kernel expands every source cell once into
 *            destination-indexed arrays.  Grids with odd nx and the two-dimensional instance always run the direct kernels.
 *   zchunk planes a block of the tiled kernels covers; 0 (default) = chosen such that the blocks fill whole waves.
 * Same results up to rounding (the kernels evaluate the same formulas in different association; the chunking matters in
 * the last place only).  ACM_EINVAL for other values. */
int acm_set_moment_kernels(acm_ctx*, int mode, int zchunk);

/* ACM_F32 only (no effect for ACM_F64).  The fp32 instance stores h_i - ref w_i and phi - ref instead of h_i and
 * phi, where ref = 0 (light) or 1 (heavy) is a reference phase: the bulk of that phase then keeps all its digits
 * (phi = 1 - 1e-4 has 3 significant digits left in fp32, its deviation -1e-4 has 7), which matters because the
 * interface normal of eq. 5 is taken from differences of phi.  Same idea as the velocity-based g of the paper,
 * which already carries g_i - w_i (eq. 12).  phase = -1 (default): acm_init takes the phase that fills most of the
 * domain (the heavy one for slabs, which must all agree); 0 / 1 force it.  Arrays crossing the ABI are unaffected.
 * ACM_ESTATE after acm_init. */
int acm_set_reference_phase(acm_ctx*, int phase);

/* Advances n >= 0 time steps (phase-field kernel, then hydrodynamic kernel, per step).
 * Asynchronous.  ACM_ESTATE before acm_init. */
int acm_step(acm_ctx*, int n);

/* CUDA graphs for launch-bound grids.  On a small grid (config 1: 32^3) a kernel is as short as its launch; acm_step
 * then replays an executable graph of 16 consecutive steps (32 kernels; the buffer parity of the two-grid layout and
 * the even/odd kernels of the in-place pattern repeat with period 2) and launches only the remaining n mod 16 steps
 * one by one.  The graph is captured on a private stream on first use and launched on the context's stream; results
 * are bit-identical to plain launches.  mode = -1 (default): automatic, for grids of at most 2^18 cells; 0: never;
 * 1: always.  Never used while acm_profile is on or on slabs.  acm_graph_replays: graph launches so far. */
int acm_set_graph(acm_ctx*, int mode);
long long acm_graph_replays(const acm_ctx*);

/* Copies out the macroscopic fields of the current time level: phi (N), u (3N, as stored by
 * the last hydrodynamic step, eq. 22) and the pressure p = p* rho(phi) c_s^2 with
 * p* = sum_i g_i (eq. 15).  [device] pointers; any may be NULL = skipped. */
int acm_fields(acm_ctx*, void* phi, void* u, void* p);

/* Total phase-field mass sum_x phi(x) (eq. 7 summed over the grid), accumulated in fp64 by a
 * deterministic two-pass block reduction.  Synchronises the stream.  total_host: [host].
 * ACM_EUNSTABLE if the sum is not finite. */
int acm_phi_mass(acm_ctx*, double* total_host);

/* Rising-bubble diagnostics of section 6.1.  The paper takes "the terminal velocity of
 * the bubbles" u_t for eq. 34 without saying how it is measured; here (reading A24) the
 * bubble is the set of cells with phi < 1/2, weighted with 1 - phi:  w = (1 - phi) [phi < 1/2]
 *   out_host[0]    V   = sum_x w
 *   out_host[1..3] X_b = sum_x w x_c / V, x_c = cell centre (i + 1/2); plain coordinates
 *   out_host[4..6] u_b = sum_x w u / V
 * fp64 accumulation, deterministic two-pass block reduction; synchronises the stream.
 * ACM_EUNSTABLE if a result is not finite (V = 0 included). */
int acm_bubble_diag(acm_ctx*, double out_host[7]);

/* Host-only helpers for the set-up and evaluation of section 6.1 (no device work):
 * acm_bubble_params solves the dimensionless groups for the lattice parameters,
 *   t_ref = sqrt(D/g_y) (eq. 33), Eo = g_y rho_H D^2/sigma (eq. 32), Re_Gr = rho_H sqrt(g_y D^3)/mu_H
 *   (eq. 31), rho* = rho_H/rho_L, mu* = mu_H/mu_L, nu = mu/rho;
 *   out_host = { g_y, sigma, nu_H, nu_L, rho_L }.  ACM_EINVAL unless every argument is > 0.
 * acm_drag_lbm = 4/3 g_y (rho_H - rho_L) D / (rho_H u_t^2) (eq. 34);
 * acm_drag_exp = [2.67^(9/10) + (16/Re_Gr)^(9/10)]^(10/9)  (eq. 35). */
int acm_bubble_params(double Re_Gr, double Eo, double D, double t_ref, double rho_H, double rho_star, double mu_star,
                      double out_host[5]);
double acm_drag_lbm(double g_y, double rho_H, double rho_L, double D, double u_t);
double acm_drag_exp(double Re_Gr);

/* Un-normalised sums behind acm_bubble_diag: { sum w, sum w x_c, sum w y_c, sum w z_c, sum w u_x, sum w u_y,
 * sum w u_z } with w = (1 - phi) [phi < 1/2] over the cells this context owns (z_c in global coordinates for a slab), so that
 * the slabs of a decomposed domain can be added up before normalising. */
int acm_bubble_sums(acm_ctx*, double out_host[7]);

/* ---- Slab decomposition along z (the paper's block decomposition with one ghost layer,
 * P:203, and its inner / outer split for communication hiding, Alg. 2 and Fig. 3) -------
 *
 * The global grid nx x ny x nz_global is cut into `nranks` slabs of consecutive z planes, one context (one
 * GPU, one process) each.  A slab stores its owned planes plus ONE ghost plane below and above:
 * every field array handed to or returned by a slab context has nz_local + 2 planes, plane 0 and plane
 * nz_local + 1 being the ghosts (arrays returned by the library leave them unspecified).
 * Periodicity / walls in z apply to the global domain; x and y are handled as before.
 *
 * The library does not communicate.  It tells the caller which byte ranges of the workspace have to travel
 * (acm_halo_plan) and lets it launch the two LB kernels on sub-ranges of planes, so that the caller
 * (paper_2012_06144_b200/slab.py: torch.distributed over NCCL/NVLink) overlaps the exchange with the kernels:
 *
 *   per step:  acm_phase_launch(0, nzl); acm_phase_commit            needs: h and phi ghosts
 *              exchange ACM_HALO_PHI (new phi) and ACM_HALO_H        (h is only needed by the NEXT phase step)
 *              acm_hydro_launch(1, nzl-1)                            inner planes: no ghost is read
 *              wait for ACM_HALO_PHI (and the g ghosts of the previous step)
 *              acm_hydro_launch(0, 1); acm_hydro_launch(nzl-1, nzl); acm_hydro_commit
 *              exchange ACM_HALO_G                                   (only needed by the NEXT hydrodynamic step)
 *
 * ACM_OPT_INPLACE and ACM_OPT_UNFUSED are not available for slabs; acm_step and acm_run_host return ACM_ESTATE. */

/* Planes [*z_begin, *z_begin + *z_count) of the global grid owned by `rank` (the first nz_global % nranks
 * slabs get one plane more).  Host only.  ACM_EINVAL unless 1 <= nranks <= nz_global, 0 <= rank < nranks. */
int acm_slab_range(int nz_global, int rank, int nranks, int* z_begin, int* z_count);
size_t acm_workspace_bytes_slab(int nx, int ny, int nz_global, int stencil_phase, int stencil_hydro, int precision,
                                int rank, int nranks);
/* acm_create_opt for the slab `rank` of `nranks`; all other arguments describe the GLOBAL problem. */
int acm_create_slab(acm_ctx** out, int nx, int ny, int nz_global, int stencil_phase, int stencil_hydro,
                    double rho_H, double rho_L, double sigma, double xi, double M, double nu_H, double nu_L,
                    const double gravity[3], unsigned wall_flags, int precision, unsigned options,
                    int rank, int nranks, void* workspace, void* cuda_stream);
/* info = { rank, nranks, first owned global plane, owned planes, allocated planes, has ghost planes (0/1) }. */
int acm_slab_info(const acm_ctx*, int info[6]);

/* What has to cross the z face `side` (0 = low z, 1 = high z) of this slab for the CURRENT buffers:
 *   ACM_HALO_H    phase populations: the e_z != 0 directions only (5 planes for D3Q15/19, 9 for D3Q27)
 *   ACM_HALO_G    hydrodynamic populations, likewise
 *   ACM_HALO_PHI  the phase field (1 plane)
 * recv = 0: the planes to SEND (this slab's outermost owned plane at that face);
 * recv = 1: the planes to RECEIVE INTO (this slab's ghost plane at that face).
 * Writes up to max_chunks (offset, bytes) pairs, offsets in bytes from the workspace base, and returns their
 * number, or -(error code).  The k-th chunk sent through a low face matches the k-th chunk received at the
 * neighbour's high face and vice versa.  Host only (valid without a GPU). */
enum { ACM_HALO_H = 0, ACM_HALO_G = 1, ACM_HALO_PHI = 2 };
int acm_halo_plan(const acm_ctx*, int what, int side, int recv, int max_chunks, size_t* offsets, size_t* bytes);

/* Peer mode of a slab: instead of reading ghost planes that an exchange has filled, the two LB kernels read the
 * planes just outside the owned range straight from the NEIGHBOUR slabs' workspaces -- the populations they pull
 * across the face and the phi stencil -- so that no population or phi plane is copied at all and the only thing
 * the ranks exchange per kernel is a completion signal.  lo_workspace / hi_workspace: [device] base pointers of the
 * workspaces the low-z / high-z neighbour contexts were created on, valid on this device: another context of the
 * same process, a CUDA-IPC mapping of another process's allocation, or a peer GPU's memory with peer access
 * enabled (NVLink).  The neighbour of the outermost slab of a periodic domain is the slab at the other end; a face
 * on a z wall needs no pointer (NULL).  All slabs must have the same height (nz_global % nranks == 0) and advance in
 * lockstep: the caller guarantees that a neighbour has finished kernel n-1 before this slab launches kernel n.
 * Both NULL switches peer mode off.  acm_get_pdfs / acm_fields(p) still read ghost planes: refresh them first. */
int acm_set_peers(acm_ctx*, void* lo_workspace, void* hi_workspace);

/* What must agree between the slabs of a decomposition in PEER mode, because a slab addresses its neighbours' arrays
 * with its OWN offsets and buffer parity: out = { workspace bytes of the layout, byte offsets of the current h, g and
 * phi buffers, hydrodynamic steps committed since acm_init, owned planes, 1 if a step is partly launched,
 * fp32 reference phase (0: fp64, 1: light, 2: heavy) }.  Host only.  The caller compares the tuples of all ranks
 * (slab.py does at set-up, after init and before it reads neighbour memory for the exports). */
int acm_state_signature(const acm_ctx*, unsigned long long out[8]);

/* Launch one LB kernel on the owned planes [z0, z1) (0 <= z0 <= z1 <= owned planes; empty range = no launch)
 * without flipping the buffers; the *_commit call flips them once all planes of the step are launched.
 * Also valid on a plain context, where acm_step(1) equals launch(0, nz), commit for both kernels.
 * The inner / outer order of Alg. 2 is guarded: ACM_ESTATE for a commit unless exactly the owned planes
 * were launched since the last commit of that kernel, for a launch that would exceed them, and for a launch of one
 * kernel while the step of the other is partly launched. */
int acm_phase_launch(acm_ctx*, int z0, int z1);
int acm_phase_commit(acm_ctx*);
int acm_hydro_launch(acm_ctx*, int z0, int z1);
int acm_hydro_commit(acm_ctx*);

/* Parity/debug export of the populations in canonical direction order and in the storage
 * convention of the paper's two LB steps: h = post-collision values at their cell (they are
 * pulled by the next phase step), g = streamed values (collide-stream-push).
 * h: [device] Q_h*N, g: [device] Q_g*N; either may be NULL. */
int acm_get_pdfs(acm_ctx*, void* h, void* g);

/* Overwrites the populations (same layout and convention as acm_get_pdfs); lets a test
 * plant an arbitrary non-equilibrium state.  Either pointer may be NULL. */
int acm_set_pdfs(acm_ctx*, const void* h, const void* g);

/* End-to-end convenience with HOST buffers: copies phi (N) and u (3N) to the device,
 * acm_init, acm_step(n), then copies phi/u/p of the final state back (NULL = skipped) and
 * synchronises the stream.  Equivalent to the calls above plus the transfers.  The result copies run on a private
 * stream behind events, each as soon as its field is final: phi right after the last phase-field kernel (it travels
 * while the last hydrodynamic kernel and the pressure export run), u after the last hydrodynamic kernel, p after its
 * export; the context's stream waits for them before the call returns. */
int acm_run_host(acm_ctx*, const void* phi_host, const void* u_host, int n,
                 void* phi_out_host, void* u_out_host, void* p_out_host);

/* Launch geometry of the two LB kernels (threads per block along x, y, z; product <= 256).
 * Optional; the defaults are tuned for B200.  ACM_ESTATE while a step is partly launched. */
int acm_set_block(acm_ctx*, int bx, int by, int bz);

/* Cells per thread of the phase-field / the hydrodynamic LB kernel: 1, or 2 = the pair kernels, in which a thread
 * updates two x-adjacent cells with 8-byte (fp32) / 16-byte (fp64) accesses wherever the pair stays aligned (own cell,
 * directions with e_x = 0) and, for fp32, Blackwell's packed fp32 arithmetic (FADD2 / FMUL2 / FFMA2: one instruction
 * per pair); 0 = the library's default for that kernel: 2 when nx is even and the kernel is fp32, or fp64 with a
 * lattice of at most 19 directions (hydrodynamic kernel: D3Q15 / D3Q19 only), else 1 (measured).  Same results up to rounding order.  A block of acm_set_block then
 * covers 2 bx cells of a row.  ACM_EINVAL for 2 with odd nx or ACM_OPT_UNFUSED. */
int acm_set_cells_per_thread(acm_ctx*, int phase, int hydro);

/* Per-kernel device timing for the roofline report.  acm_profile(ctx, 1) makes every later
 * acm_step record CUDA events on the stream around each of its two kernels (and drops earlier
 * records; the events are created before the first kernel of the call, not between kernels);
 * acm_profile(ctx, 0) switches that off.  acm_profile_read synchronises the stream,
 * returns the summed durations in milliseconds of the phase-field and the hydrodynamic kernel
 * and the number of steps they cover, and clears the records.  Pointers are [host], may be NULL. */
int acm_profile(acm_ctx*, int enable);
int acm_profile_read(acm_ctx*, double* phase_ms, double* hydro_ms, long long* steps);

/* Number of kernels this context has launched so far (bench.py's gpu_launches). */
long long acm_launch_count(const acm_ctx*);

void acm_destroy(acm_ctx*);

/* Thread-local description of the last error; never NULL. */
const char* acm_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* ACM_H_ */

/*
 * afid.h -- C ABI of the B200-native AFiD pressure-correction (projection) step.
 *
 * What the library computes (paper = arXiv 1705.01423, "P:L<n>" = line n of PAPER.md):
 * one projection of a provisional, non-solenoidal velocity (u*, v*, w*) onto the discretely
 * divergence-free fields of a staggered, conservative, second-order finite-difference grid
 * (Fig. 1) by the fractional-step method: solve the Poisson equation
 * D G phi = D u* for the pressure correction phi, then u = u* - G phi.  The solve
 * is the direct method of P:L99-L114: Fourier transforms in the two periodic directions
 * (y, z) with modified wavenumbers, one tridiagonal system in the wall-normal direction x
 * per (ky, kz) mode, inverse transforms.  Readings of everything the paper leaves open
 * (metrics, the singular mean mode, p = phi) are listed in DESIGN.md, section "Readings".
 *
 * Grid.  nx cells in x between the walls xc[0] and xc[nx] (xc: nx+1 strictly increasing
 * face coordinates, possibly stretched); ny, nz uniform periodic cells over lengths
 * Ly, Lz.  Arrays are C-ordered [i][j][k], k (z) fastest, fp64, 64-bit indexing:
 *   u : (nx+1)*ny*nz  wall-normal velocity on x-faces (planes 0 and nx are the walls)
 *   v :  nx   *ny*nz  y-velocity on y-faces
 *   w :  nx   *ny*nz  z-velocity on z-faces
 *   p :  nx   *ny*nz  pressure correction phi at cell centres (output only)
 *
 * All work runs in hand-written sm_100a CUDA kernels; there is no CPU or library (cuFFT)
 * fallback: an unsupported size or a missing device is an error.
 *
 * Threading: a plan may be used by one host thread / one stream at a time.  Functions never
 * synchronise the device unless stated.
 */
#ifndef AFID_H_
#define AFID_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct afid_plan afid_plan; /* opaque; owned by the library */

/* Error codes (negative).  afid_last_error() returns a message for the calling thread. */
#define AFID_OK 0
#define AFID_ERR_NULL (-1)             /* a required pointer is NULL                               */
#define AFID_ERR_ALIGN (-2)            /* a device pointer is not 16-byte aligned                  */
#define AFID_ERR_UNSUPPORTED_SIZE (-3) /* nx, ny or nz outside what the kernels are built for     */
#define AFID_ERR_GRID (-4)             /* xc not finite / not strictly increasing, or Ly, Lz <= 0  */
#define AFID_ERR_NOMEM (-5)            /* device or host allocation failed                         */
#define AFID_ERR_CUDA (-6)             /* a CUDA runtime call or kernel launch failed              */

/*
 * afid_plan_create -- build a plan for an nx x ny x nz grid on the CURRENT CUDA device.
 *   nx      cells in x, 2 <= nx <= afid_max_nx()
 *   ny, nz  periodic cells; ny and nz/2 must be lengths the FFT kernels are instantiated
 *           for (afid_fft_length_supported, afid_fft_half_length_supported):
 *             ny   a multiple of 8 in 8..4096 of the form 2^a 3^b (b <= 4), or 5 2^a (40..2560);
 *             nz/2 an even number in 8..1536 of the form 2^a 3^b (b <= 4; up to 1024 for pure powers of two
 *                  and 1536 = 3 2^9, i.e. nz <= 3072), or 5 2^a (40..1280)
 *           (the paper's grids, Tables 2-4: 768 x 768 x 1296, 1280 x 1024 x 256, 2048 x 3072 x 3072 slabs)
 *   xc      HOST pointer, nx+1 face coordinates (copied; caller keeps ownership)
 *   Ly, Lz  periodic box lengths (> 0)
 * The plan owns: reciprocal metrics, tridiagonal coefficients a_i, c_i, modified
 * wavenumbers 2(1-cos(2 pi k/n))/Delta^2, twiddle tables, and two device work
 * arrays of nx*ny*(nz/2+1) complex doubles each.  Synchronous (allocates and uploads).
 * Returns NULL on failure (see afid_last_error / afid_last_error_code).
 */
afid_plan* afid_plan_create(int nx, int ny, int nz, const double* xc, double Ly, double Lz);

/*
 * afid_project -- enqueue one projection step on `stream` (a cudaStream_t, may be NULL for
 * the legacy default stream).  u, v, w, p are DEVICE pointers, 16-byte aligned, laid out as
 * above, owned by the caller.  u, v, w are updated in place (the two wall planes of u are
 * read, never written: Neumann condition on phi); p is overwritten with phi, whose
 * dx-weighted mean is zero.  Steps (paper step numbers):
 *   1  divergence                        3+5  forward transforms in z then y
 *   7  tridiagonal solves in x           9+11 inverse transforms in y then z
 *   correction u -= G phi, p = phi
 * (steps 2,4,6,8,10,12, the pencil transposes, are folded into the kernels' tile loads).
 * Returns AFID_OK or a negative code.  Validation is synchronous; the kernels are only
 * enqueued, so execution errors surface at the caller's next synchronisation.
 * The call only enqueues kernels (and, with timing enabled, event records) on `stream`, so it may be captured
 * in a CUDA graph and replayed.
 * NaN/Inf in the inputs propagate.  The compatibility condition (zero net wall flux) is
 * not checked; it holds identically when u vanishes on both wall planes.
 */
int afid_project(afid_plan* plan, double* u, double* v, double* w, double* p, void* stream);

/*
 * afid_max_cfl -- SURVEY.md 8(f3): the maximum CFL number of a velocity field, the routine the paper
 * prints in full (Listing 1 "CalcMaxCFL"):
 *     cfl = max( 1e-8, max over cells (i,j,k) of
 *                0.5 * ( |w(i,j,k) + w(i,j,k+1)| / dz + |v(i,j,k) + v(i,j+1,k)| / dy + |u(i,j,k) + u(i+1,j,k)| / dx_i ) )
 * with periodic wrap in j and k (the listing's dz, dy, udx3m are AFiD's inverse spacings).
 * u, v, w: DEVICE pointers laid out as for afid_project (read only, 16-byte aligned); cfl: DEVICE pointer to
 * one double (8-byte aligned), overwritten.  Two kernels are enqueued on `stream`; no host synchronisation.
 * Typically called on the projected field to pick the next time step.  Returns AFID_OK or a negative code.
 */
int afid_max_cfl(afid_plan* plan, const double* u, const double* v, const double* w, double* cfl, void* stream);

/*
 * afid_project_cfl -- SURVEY.md 8(f3), fused form: afid_project, and the maximum CFL number (afid_max_cfl's
 * definition, Listing 1) of the CORRECTED field into *cfl, taken inside the correction launch:
 * the corrected u, v, w are reduced while they are still in L2 instead of being read back from HBM by a
 * second pass (24 B per point).  Same arguments as afid_project plus cfl (DEVICE pointer to one double,
 * 8-byte aligned, overwritten).  u, v, w, p come out bit-identical to afid_project's, and *cfl bit-identical
 * to afid_max_cfl on them.  Enqueue only (one memset, five kernels + two small ones); capturable in a CUDA
 * graph.  Unsharded plans only; not available with afid_plan_set_pipeline.
 */
int afid_project_cfl(afid_plan* plan, double* u, double* v, double* w, double* p, double* cfl, void* stream);
/* afid_cfl_schedule -- HOST arithmetic only (no device, no plan), for tests of the fused launch's schedule: ticket t
 * corrects item t = lines 4 jg .. 4 jg + 3 of plane i (the order of the correction kernel) and then reduces the
 * cells of item t - lag, lines [line_lo, line_hi] (one line down) plus extra_line (ny - 1 for the last group, else
 * -1), after the items deps[0..4] (-1 = none) have been corrected.  ny must be a multiple of 4. */
int afid_cfl_schedule(int nx, int ny, int item, int* i, int* jg, int* line_lo, int* line_hi, int* extra_line, int* deps);

/*
 * afid_plan_set_accumulate -- SURVEY.md 8(f3): choose what afid_project does with p.
 *   on = 0 (default)  p  = phi   (p is output only; its dx-weighted mean is zero; R6)
 *   on = 1            p += phi   (the "delta form" pressure update of the fractional step, P:L91, P:L116;
 *                                 phi then goes through a work array and p is read and written by the
 *                                 correction kernel: 16 more bytes per point)
 * The velocity correction is the same in both modes.  Returns AFID_OK or a negative code.
 */
int afid_plan_set_accumulate(afid_plan* plan, int on);

/*
 * afid_xsolve_* -- batched REAL tridiagonal solves in the wall-normal direction on a field in
 * physical space, the implicit (Crank-Nicolson) wall-normal viscous step of the time integrator (
 * "batched tridiagonal solvers").  For every (j,k) column of f[i][j][k] (layout of v, w, p), in place:
 *     -a_i x_{i-1} + (a_i + c_i + lam_i) x_i - c_i x_{i+1} = f_i ,   i = 0..nx-1   (a_0 and c_{nx-1} are ignored)
 * i.e. (I - theta L_x) x = r scaled by 1/theta, with L_x x = a_i x_{i-1} - (a_i + c_i) x_i + c_i x_{i+1} and
 * lam_i = 1/theta (+ the Dirichlet ghost-cell terms in the wall rows).  The paper does not print the
 * coefficients of its scheme (they are in its Refs [19],[27]), so they are the caller's: HOST arrays of nx
 * doubles, a_i >= 0, c_i >= 0, lam_i > 0 (an M-matrix: the solve is cancellation-free), copied at create.
 * afid_xsolve_create is synchronous and returns NULL on failure; afid_xsolve_apply only enqueues one kernel
 * (the x-solve kernel of afid_project, two neighbouring k columns per complex lane) on `stream`;
 * f: DEVICE, nx*ny*nz doubles, 16-byte aligned.  The plan must outlive the handle.
 */
typedef struct afid_xsolve afid_xsolve;
afid_xsolve* afid_xsolve_create(afid_plan* plan, const double* a, const double* c, const double* lam);
int afid_xsolve_apply(afid_xsolve* h, double* f, void* stream);
int afid_xsolve_destroy(afid_xsolve* h);

/*
 * afid_plan_set_pipeline -- run the two transform sweeps of afid_project plane-pipelined, so that their
 * intermediates are handed from kernel to kernel inside the 126 MB L2 instead of through HBM (the paper's
 * motivation for its hand-written local transposes, and for caring about bandwidth at all).
 *   planes_per_batch > 0: the forward sweep (divergence + z transform, then y transform) and the inverse
 *       sweep (inverse y transform, inverse z transform, correction) are launched in batches of that many
 *       y-z planes on plan-owned streams, forked from and joined back to `stream` with events: the
 *       kernels of batch b overlap those of batch b-1, and the z-transformed (y-transformed) plane goes
 *       through a rotating buffer of `rotation` batches (2 <= rotation <= 7; planes_per_batch a multiple
 *       of 2 where the inverse y transform handles two planes per CTA; planes_per_batch * rotation <= nx).
 *   planes_per_batch <= 0: one launch per kernel over all planes (six launches; the default).
 * Results are bit-identical in both modes.  Still capturable in a CUDA graph (fork/join by events).
 * With timing enabled only the three sweeps are timed (afid_plan_num_timed).
 * afid_plan_set_l2_hints -- bit mask of L2 eviction-priority hints the kernels attach to their accesses:
 *   1 streamed loads (u, v, w, spectra read once) evict-first      2 intermediates (B, D) evict-last
 *   4 loads of the intermediates evict-first                       8 streamed stores evict-first
 *   32 afid_project_cfl runs its two-CTAs-per-SM kernel variant (in that kernel bit 2 also makes the corrected
 *      lines evict-last and bit 4 drops the evict-first hint of the uncorrected loads): measurement switches
 * Default 0.  Hints change timing only, never results.
 */
int afid_plan_set_pipeline(afid_plan* plan, int planes_per_batch, int rotation);
int afid_plan_set_l2_hints(afid_plan* plan, int mask);

/*
 * afid_shard_* -- the projection sharded over `nranks` GPUs, one process per GPU.  The paper
 * distributes the solver with pencils and SIX all-to-all transposes per projection, staged through the host
 * (P:L103-L114); with one address space per GPU and NVLink/NVSwitch between them two
 * exchanges are enough:
 *   x-slabs       rank r owns the planes [xs, xe) = [nx r/R, nx (r+1)/R) for the divergence, both transforms and the
 *                 correction (a y-z plane is local to one rank);
 *   kz partition  rank r owns the modes kz in [ks, ke) = [nzh r/R, nzh (r+1)/R), nzh = nz/2+1, for the x-solves
 *                 (all nx rows of a system are local to one rank);
 *   exchange 1    forward spectrum: slabs -> kz partition;   exchange 2   solved spectrum: kz partition -> slabs;
 *   halo          one plane of phi from the rank below (for the first u plane of the slab); the caller supplies
 *                 the slab's upper halo plane of u (plane xe, the first plane of the rank above or the wall).
 * The library does the arithmetic and the re-layouts; the exchanges themselves are the caller's (the Python binding
 * uses torch.distributed all_to_all_single over NCCL, send/recv for the halo): afid_shard_layout says how many
 * complex elements go to / come from each peer and at which offsets of the buffers afid_shard_buffers returns.
 * One projection on rank r, all calls enqueue on `stream`:
 *     afid_shard_forward(plan, u, v, w)          u: (xe-xs+1)*ny*nz (slab + upper halo plane), v, w: (xe-xs)*ny*nz
 *     exchange 1   (all-to-all, counts/offsets of afid_shard_layout(..., phase 1, ...))
 *     afid_shard_solve(plan)
 *     exchange 2   (phase 2)
 *     afid_shard_inverse(plan, p)                p: (xe-xs)*ny*nz <- phi of the slab
 *     halo         p_halo <- last plane of p of rank r-1 (ny*nz doubles)
 *     afid_shard_correct(plan, u, v, w, p, p_halo)      p_halo ignored (may be NULL) on rank 0
 * u, v, w, p are this rank's slabs (DEVICE, same layout as afid_project); the slab's own planes of u, v, w are
 * updated in place (the halo plane of u is read only).  The result equals afid_project on the whole grid bit for
 * bit: the same kernels run on the same lines and systems.  afid_max_cfl on a sharded plan returns the slab's
 * maximum (the caller all-reduces it).  afid_project, the stage taps, afid_xsolve_* and the accumulate
 * mode need an unsharded plan.  nranks <= 64, nranks <= nx, nranks <= nz/2+1.
 * afid_shard_bounds / afid_shard_layout are host arithmetic only (usable without a device).
 */
afid_plan* afid_shard_plan_create(int nx, int ny, int nz, const double* xc, double Ly, double Lz, int rank, int nranks);
int afid_shard_bounds(int n, int nranks, int rank, int* lo, int* hi);   /* part `rank` of n items: [n rank/nranks, n (rank+1)/nranks) */
int afid_shard_layout(int nx, int ny, int nz, int nranks, int rank, int phase, long long* send_count, long long* send_off,
                      long long* recv_count, long long* recv_off);       /* HOST arrays of nranks entries each */
int afid_shard_buffers(afid_plan* plan, int phase, void** send, void** recv);
int afid_shard_info(const afid_plan* plan, int* rank, int* nranks, int* xs, int* xe, int* ks, int* ke);
int afid_shard_forward(afid_plan* plan, const double* u, const double* v, const double* w, void* stream);
int afid_shard_solve(afid_plan* plan, void* stream);
int afid_shard_inverse(afid_plan* plan, double* p, void* stream);
int afid_shard_correct(afid_plan* plan, double* u, double* v, double* w, double* p, const double* p_halo, void* stream);

/* afid_plan_destroy -- free the plan's device and host memory.  NULL is a no-op.
 * The caller must have synchronised any stream still using the plan. */
int afid_plan_destroy(afid_plan* plan);

/* Device bytes held by the plan (work arrays + tables). */
size_t afid_plan_workspace_bytes(const afid_plan* plan);

/* Number of kernel launches one afid_project call enqueues (for launch accounting). */
int afid_plan_num_launches(const afid_plan* plan);

/*
 * Per-kernel device timing, for the roofline report.  With timing enabled afid_project
 * records a CUDA event on `stream` before and after each of its kernels (no host sync).
 * afid_plan_kernel_times synchronises on the last recorded event and writes the duration in
 * milliseconds of each kernel of the most recent afid_project call into ms[0..n-1]
 * (HOST pointer, n <= afid_plan_num_timed); afid_plan_kernel_name gives their names.
 */
int afid_plan_enable_timing(afid_plan* plan, int on);
int afid_plan_num_timed(const afid_plan* plan); /* entries afid_plan_kernel_times writes: 6 kernels, or 3 sweeps when pipelined */
int afid_plan_kernel_times(afid_plan* plan, float* ms, int n);
const char* afid_plan_kernel_name(const afid_plan* plan, int k);

/*
 * Stage taps, for stage-wise parity tests (same kernels as afid_project, run separately):
 *   afid_stage_forward:  u,v,w -> spectrum of -(div u)/(ny*nz), written to `spec`
 *                        (DEVICE, nx*(nz/2+1)*ny complex doubles, layout [i][kz][ky]).
 *   afid_stage_solve:    spec ([i][kz][ky], in place) <- solution of the x-systems.
 * Both enqueue on `stream` and use the plan's work arrays.
 */
int afid_stage_forward(afid_plan* plan, const double* u, const double* v, const double* w,
                       double* spec, void* stream);
int afid_stage_solve(afid_plan* plan, double* spec, void* stream);

/* 1 if the y-direction FFT kernels are instantiated for complex length n (ny must satisfy this). */
int afid_fft_length_supported(int n);
/* 1 if the z-direction (real-data) FFT kernels are instantiated for half length n (nz/2 must satisfy this). */
int afid_fft_half_length_supported(int n);
/* Largest nx the tridiagonal kernel supports. */
int afid_max_nx(void);

const char* afid_last_error(void);  /* thread-local message of the last failure ("" if none) */
int afid_last_error_code(void);     /* thread-local code of the last failure                 */
const char* afid_version(void);

#ifdef __cplusplus
}
#endif
#endif /* AFID_H_ */

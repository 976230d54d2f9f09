/*
 * dks_poisson.h -- C ABI of the B200-native open-boundary FFT Poisson solver.
 *
 * The operation (arXiv:1509.07685, "The Dynamical Kernel Scheduler - Part 1"):
 *   PAPER.md:119-122, section 3.1.1, Eq. (2):
 *       phi[i,j,k] = hx*hy*hz * sum_{i',j',k'} rho[i',j',k'] * G((i-i')hx, (j-j')hy, (k-k')hz)
 *   computed as (section 3.1.1)
 *       phi = hx*hy*hz * FT^-1{ FT{rho} (x) FT{G} }
 *   on Hockney's doubled grid 2Mx x 2My x 2Mz (section 3.1), with
 *       G(u,v,w) = 1 / (4*pi*eps0*sqrt(u^2+v^2+w^2))        (the 1/(4 pi eps0) follows
 *   from the PDE laplace(phi) = -rho/eps0 at PAPER.md:104; eps0 = 8.8541878128e-12 F/m).
 *   The paper's GPU implementation (section 3.1.2) has "separate kernels to calculate
 *   the Greens function and perform the multiplication" around a library FFT; here every step is a
 *   hand-written sm_100a kernel and padding, multiplication, cropping and scaling are fused into
 *   the FFT passes.
 *
 * Conventions
 *   - mesh n = (nx, ny, nz) = the paper's (Mx, My, Mz); every n must be a power of two in [8, 1024]
 *     (Table 1, uses powers of two only).
 *   - rho, phi: DEVICE pointers, contiguous fp64, x fastest: linear index (k*ny + j)*nx + i, i.e. a
 *     [nz][ny][nx] array; 16-byte aligned.  phi in volts for rho in C/m^3 and h in metres.
 *   - G(0,0,0) defaults to G at r0 = min(hx,hy,hz)/2 (the paper is silent; reading A2).
 *   - All calls return DKS_OK (0) or a negative dks_status; nothing throws or aborts across the ABI.
 *     dks_last_error() returns a thread-local, NUL-terminated message for the last failure.
 *   - A plan is a host object owning host metadata and device twiddle tables.  It is not re-entrant:
 *     one solve in flight per plan.
 *   - There is no CPU fallback.  Without a compute-capability 10.x device every compute entry point
 *     returns DKS_ERR_UNSUPPORTED_DEVICE / DKS_ERR_CUDA.
 */
#ifndef DKS_POISSON_H
#define DKS_POISSON_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum dks_status {
    DKS_OK = 0,
    DKS_ERR_INVALID_ARG = -1,        /* NULL pointer, n not a power of two in [8,1024], h <= 0 or not finite */
    DKS_ERR_UNSUPPORTED_DEVICE = -2, /* current device is not compute capability 10.x                      */
    DKS_ERR_WORKSPACE_TOO_SMALL = -4,/* dks_poisson_set_workspace: bytes < dks_poisson_workspace_bytes     */
    /* -3 is not used: SURVEY.md section 8(b) lists a NO_WORKSPACE status; a plan without a workspace allocates its own in
     * dks_greens_setup, so the only way to meet that state is to call an entry point before the set-up, and that is
     * reported as DKS_ERR_NOT_SETUP (dks_field_at_particles, dks_poisson_shard_buffers, dks_poisson_set_peers). */
    DKS_ERR_NOT_SETUP = -5,          /* dks_poisson_solve before dks_greens_setup (or after a spacing change) */
    DKS_ERR_CUDA = -6                /* a CUDA runtime call failed; see dks_last_error()                   */
} dks_status;

typedef struct dks_poisson_plan dks_poisson_plan;   /* opaque */

/* Creates a plan for an nx x ny x nz mesh (the paper's Mx x My x Mz) with spacings hx, hy, hz [m]
 * (the mesh is fitted to the bunch, so h is a per-time-step quantity).  The plan plays the role of the
 * device-side state that DKS keeps between the calls of Fig. 2.  Host-only: validates the
 * arguments and computes the twiddle tables on the host; touches no device.  Returns NULL on
 * failure (dks_last_error() says why). */
dks_poisson_plan *dks_poisson_plan_create(int nx, int ny, int nz, double hx, double hy, double hz);

/* Frees the plan, its device tables and (if plan-owned) its workspace (Fig. 2's freeMemory).  Caller-owned
 * workspaces are left alone.  The caller makes sure no solve of this plan is still running.  NULL is allowed. */
void dks_poisson_plan_destroy(dks_poisson_plan *plan);

/* Step a0 ("separate kernels to calculate the Greens function"):
 * builds G on the octant of the doubled grid (mirror rule i' = min(i, 2n-i)), transforms it
 * (the transform of the even extension is real and even, so only the (nx+1)(ny+1)(nz+1) octant is
 * kept) and folds the factor hx*hy*hz/(8 nx ny nz) in.  Allocates the plan-owned workspace on first
 * use if none was attached.  Asynchronous on the plan's setup stream (default: the legacy default
 * stream); a later dks_poisson_solve on another stream is ordered after it by an event. */
int dks_greens_setup(dks_poisson_plan *plan);

/* The hot path: phi = hx hy hz FT^-1{FT{rho} (x) FT{G}} cropped to the mesh.
 * rho_dev, phi_dev: device pointers as described above; rho_dev is only read; phi_dev may alias
 * rho_dev.  stream: a cudaStream_t (NULL = legacy default stream).  Asynchronous and stream-ordered:
 * no host synchronisation, no allocation; CUDA-graph capturable (a captured solve is not ordered against later
 * dks_greens_setup calls: the caller orders graph replays and rebuilds).  Launches P1, then P2-P3-P4 once per
 * slab of kz planes (dks_poisson_set_slab_planes; default: one slab), then P5: 2 + 3 * ceil((nz+1)/slab) kernels.
 * Errors: DKS_ERR_INVALID_ARG (NULL or misaligned pointer), DKS_ERR_NOT_SETUP, DKS_ERR_CUDA. */
int dks_poisson_solve(dks_poisson_plan *plan, const double *rho_dev, double *phi_dev, void *stream);

/* Several independent meshes of the same shape and spacing in one call (e.g. neighbouring bunches, PAPER.md:140
 * ref. [27]): rho_dev and phi_dev hold nbatch meshes back to back ([nbatch][nz][ny][nx]).
 * Every pass processes the whole batch in one launch (still five launches), so small meshes are no longer
 * launch-latency bound and all meshes share one Green's transform.  nbatch <= dks_poisson_set_max_batch, which
 * sizes the workspace (A and B scale with it; default 1) and must be called before the workspace is attached /
 * before dks_greens_setup.  Needs the default pipeline (no slabs).  Same stream semantics as
 * dks_poisson_solve; phi_dev may alias rho_dev. */
int dks_poisson_set_max_batch(dks_poisson_plan *plan, int nbatch);
int dks_poisson_solve_batch(dks_poisson_plan *plan, const double *rho_dev, double *phi_dev, int nbatch, void *stream);

/* Same solve with HOST buffers (the end-to-end path of the paper: rho is copied to
 * the device and phi back every step).  rho_host/phi_host: host pointers ([nz][ny][nx] fp64; pinned
 * memory recommended).  = dks_poisson_solve_host_async followed by dks_poisson_host_sync: the copies run on
 * plan-owned streams, the solve on `stream`, and the call returns when phi_host is complete.  Work issued on
 * `stream` afterwards is ordered after the solve, not after the copy-out (the host has waited for that).
 * The staging buffers are part of the workspace. */
int dks_poisson_solve_host(dks_poisson_plan *plan, const double *rho_host, double *phi_host, void *stream);

/* The same without the final synchronisation, so that consecutive steps overlap (PAPER.md:132 overlaps the rho
 * transfer with device work through streams): the copy-in of call i+1 and the copy-out of call i-1 run on
 * plan-owned streams beside the solve of call i, which runs on `stream`; three staging meshes take turns (a slot is busy from its copy-in to its copy-out).  Every
 * call still moves its own rho and phi.  phi_host of a call is complete after dks_poisson_host_sync (which
 * waits for every copy-out issued so far); rho_host must stay unchanged until then.  Pinned host memory is
 * needed for the overlap.  Not capturable in a CUDA graph. */
int dks_poisson_solve_host_async(dks_poisson_plan *plan, const double *rho_host, double *phi_host, void *stream);
int dks_poisson_host_sync(dks_poisson_plan *plan);

/* One time step exactly as the paper runs it (Fig. 5: "CUDA streams are used to overlap the transfer of
 * the rho field to the GPU and the calculation of the Greens function"; the spacings change every step):
 * dks_poisson_set_spacing(hx, hy, hz), then the Green's rebuild (step a0) on the setup stream -- a plan-owned stream
 * unless dks_poisson_set_stream gave one that differs from `stream` -- concurrently with the host-to-device copy of
 * rho on the copy-in stream; the solve on `stream` waits for both, the copy-out follows on the copy-out stream.  The
 * rebuild of step i+1 is ordered after P3 of step i (the only reader of the Green's transform), so it also overlaps
 * P4, P5 and the copy-out of step i.  Same buffer rules as dks_poisson_solve_host_async; finish with
 * dks_poisson_host_sync. */
int dks_poisson_step_host_async(dks_poisson_plan *plan, double hx, double hy, double hz, const double *rho_host,
                                double *phi_host, void *stream);

/* Changes the mesh spacings (they are time dependent).  Host-only.  Invalidates the Green's
 * transform: call dks_greens_setup again before the next solve (DKS_ERR_NOT_SETUP otherwise). */
int dks_poisson_set_spacing(dks_poisson_plan *plan, double hx, double hy, double hz);

/* Overrides G(0,0,0), which PAPER.md:117 leaves undefined (G = 1/r is singular there; reading A2);
 * NaN restores the default rule G(r0), r0 = min(hx,hy,hz)/2.  Host-only.  Invalidates the Green's transform. */
int dks_poisson_set_g0(dks_poisson_plan *plan, double g0_or_nan);

/* Bytes of device workspace the plan needs (buffer A, the Green's octant, the three host-path staging
 * meshes unless switched off, one slab of B).  "Memory management is left up to the user": the caller may allocate it
 * (Fig. 2's allocateMemory) and attach it with dks_poisson_set_workspace.  Host-only. */
size_t dks_poisson_workspace_bytes(const dks_poisson_plan *plan);

/* The host path (dks_poisson_solve_host*, dks_poisson_step_host_async) stages rho / phi in three mesh-sized buffers inside the
 * workspace (3 x 8 nx ny nz bytes: 403 MB at 256^3).  A caller whose meshes stay on the device (PAPER.md:160 is the argument for
 * that) can leave them out: enabled = 0 shrinks dks_poisson_workspace_bytes() accordingly and makes the host-path calls fail
 * with DKS_ERR_NOT_SETUP.  Default: enabled.  Call it before the workspace is attached / before dks_greens_setup
 * (DKS_ERR_INVALID_ARG afterwards).  Sharded plans never carry the staging buffers and refuse the host path.  Host-only. */
int dks_poisson_set_host_staging(dks_poisson_plan *plan, int enabled);

/* Attaches caller-owned device memory (e.g. a torch tensor) as the workspace (Fig. 2);
 * 256-byte aligned, at least dks_poisson_workspace_bytes() (else DKS_ERR_WORKSPACE_TOO_SMALL).  The caller keeps
 * ownership and must keep it alive.  Invalidates the Green's transform.  Without it dks_greens_setup allocates a
 * plan-owned workspace on first use. */
int dks_poisson_set_workspace(dks_poisson_plan *plan, void *dev_ptr, size_t bytes);

/* P2, P3 and P4 work on independent kz planes of the half-spectrum (kz = 0..nz).  They are launched
 * slab by slab -- `planes` consecutive kz planes at a time -- so that the buffer B between them
 * ([planes][2ny][nx] complex) is a scratch that stays in the L2 cache instead of going through HBM.
 * planes = 0 restores the automatic choice, which is one slab of all nz+1 planes (measured: every slab boundary
 * costs more than the L2 residency saves); planes = nz+1 is the same unslabbed pipeline.  Changes dks_poisson_workspace_bytes(); call it before attaching a workspace / before
 * dks_greens_setup (afterwards it fails with DKS_ERR_WORKSPACE_TOO_SMALL if the workspace cannot
 * hold the new slab).  Switches per-pass profiling off.  dks_poisson_slab_planes returns the
 * current value. */
int dks_poisson_set_slab_planes(dks_poisson_plan *plan, int planes);
int dks_poisson_slab_planes(const dks_poisson_plan *plan);

/* Stream used by dks_greens_setup (default NULL = legacy default stream): "GPU streams are used" for asynchronous
 * work, here to overlap the Green's rebuild with the rho transfer.  Solves on other
 * streams are ordered after the rebuild, and the next rebuild after their P3, by plan-owned events.  Host-only. */
int dks_poisson_set_stream(dks_poisson_plan *plan, void *stream);

/* Per-pass timing.  slots > 0: dks_poisson_solve records CUDA events on its stream around each of
 * its launches (still asynchronous) and keeps those of the last `slots` solves (slots <= 256);
 * slots = 0 switches it off.  dks_poisson_pass_times waits for the recorded solves and writes up to
 * `count` durations in milliseconds (pass order P1..P5, summed over the slabs), each the mean over the
 * recorded solves;
 * returns the number of passes written or a negative status. */
int dks_poisson_set_profiling(dks_poisson_plan *plan, int slots);
int dks_poisson_pass_times(dks_poisson_plan *plan, float *ms_out, int count);

/* Facts about the plan, for benchmarks and tests. */
int    dks_poisson_launches_per_solve(const dks_poisson_plan *plan);   /* kernels launched by one solve   */
double dks_poisson_model_bytes(const dks_poisson_plan *plan, int pass); /* algorithmic HBM bytes of pass 1..5; pass 0 = whole solve (DESIGN.md model M3) */
const char *dks_poisson_pass_name(const dks_poisson_plan *plan, int pass); /* kernel variant used for pass 1..5 */

/* Copies the Green's octant (real, [(nz+1)][(ny+1)][(nx+1)], scale folded in) to a host buffer of
 * (nx+1)(ny+1)(nz+1) doubles; synchronises.  For tests. */
int dks_poisson_copy_greens_hat(dks_poisson_plan *plan, double *host_out);

/* ---- The steps adjacent to the solve, on the device ------------------------------------------
 * OPAL's particles come "with the respective interpolation operators" (IPPL); moving rho and
 * phi between host and device costs "up to 55 %" of the run.  With the deposit before and the field evaluation after the
 * solve on the device, only particle data (or nothing, if the particles live there) crosses the host link.  The paper
 * gives no formulas; readings F1-F4: node (i,j,k) sits at origin + (i hx, j hy, k hz) with the plan's CURRENT
 * spacings; cloud-in-cell (trilinear) weights; a particle is dropped unless 0 <= (X - ox)/hx < nx - 1 (likewise y, z);
 * E = -grad(phi) by second-order differences (central inside, one-sided second order at the ends; every extent >= 8).
 * All pointers are DEVICE pointers to contiguous fp64; meshes are [nz][ny][nx]; particle arrays hold np entries (SoA).
 * Asynchronous on `stream`, no allocation, no synchronisation; none of them needs dks_greens_setup. */

/* rho[node] = sum_p q_p w_p(node) / (hx hy hz) (C/m^3 for q in C).  rho is zeroed first (on `stream`).  The sums are
 * fp64 atomics: order-free, so equal to a sequential sum only to a few ulp of each node's total. */
int dks_deposit_cic(dks_poisson_plan *plan, const double *x_dev, const double *y_dev, const double *z_dev, const double *q_dev,
                    long long np, double ox, double oy, double oz, double *rho_dev, void *stream);

/* (ex, ey, ez) = -grad(phi) [V/m]; the outputs must not alias phi. */
int dks_gradient(dks_poisson_plan *plan, const double *phi_dev, double *ex_dev, double *ey_dev, double *ez_dev, void *stream);

/* Field at the particles: trilinear interpolation of (ex, ey, ez) with the deposit's weights; 0 for dropped particles. */
int dks_gather_field(dks_poisson_plan *plan, const double *ex_dev, const double *ey_dev, const double *ez_dev,
                     const double *x_dev, const double *y_dev, const double *z_dev, long long np, double ox, double oy, double oz,
                     double *epx_dev, double *epy_dev, double *epz_dev, void *stream);

/* dks_gradient followed by dks_gather_field in one call, for the per-step use: the field at the particles
 * straight from phi, readings F3 + F4, same results as the two calls.  The node field is not returned; it lives for the duration
 * of the call in the plan's buffer B, interleaved (ex, ey, ez per node in one 32-byte record, so the gather needs one 256-bit load
 * per node).  Needs the plan's workspace (dks_poisson_set_workspace or a previous dks_greens_setup; DKS_ERR_NOT_SETUP otherwise)
 * and the unslabbed, unsharded pipeline (DKS_ERR_INVALID_ARG otherwise); must not run concurrently with a solve of the same
 * plan (both use B).  Asynchronous on `stream`. */
int dks_field_at_particles(dks_poisson_plan *plan, const double *phi_dev, const double *x_dev, const double *y_dev,
                           const double *z_dev, long long np, double ox, double oy, double oz, double *epx_dev, double *epy_dev,
                           double *epz_dev, void *stream);

/* ---- The field at the particles without any device allocation ---------------------------------------------------------------
 * Same operation and same results as dks_field_at_particles (gradient of phi by second-order differences, readings F3 + F4,
 * then trilinear interpolation to the particles), for callers that cannot allocate device memory: no plan
 * is needed (creating and using a plan calls cudaMalloc for its tables and, unless one is attached, its workspace).  Who
 * that is: a time-step loop whose other streams a cudaMalloc / cudaFree would stall, because both synchronise the device; a
 * host program whose own pool already holds all device memory, so that any further cudaMalloc fails; a component that is
 * only ever handed device pointers and has no allocator of its own.
 *
 * The node field (one 32-byte record per node) goes into an array that is part of the library image: 8 MiB of device
 * memory, held by every GPU on which the library's CUDA module is loaded until the process exits.  Hence the limit
 * nx * ny * nz <= DKS_STATIC_FIELD_MAX_NODES (64 x 64 x 64, 128 x 64 x 32, ...); a larger mesh is refused with
 * DKS_ERR_INVALID_ARG and a message naming the limit.  nx, ny, nz: powers of two in [8, 1024] as for a plan; hx, hy, hz > 0.
 * phi_dev [nz][ny][nx], the particle arrays (np entries each) and the three outputs are DEVICE pointers the caller owns;
 * the call itself never calls cudaMalloc, cudaFree or any library routine that allocates.
 *
 * First call on a device: looks up the device address of the array (cudaGetSymbolAddress, with that device current) and the
 * SM count, and keeps them for later calls.  Make that first call outside any stream capture.  Later calls only launch two
 * kernels on `stream` (asynchronous, no synchronisation).
 *
 * All calls on one device share the one array.  It keeps whatever the last call wrote; that is harmless, because a call
 * writes the record of every node of its mesh before it reads any.  But two calls that are in flight on the same GPU at
 * the same time (different streams, or different host threads) overwrite each other's records: the caller must order
 * them, e.g. by issuing them on one stream. */
#define DKS_STATIC_FIELD_MAX_NODES (1 << 18)
int dks_field_at_particles_static(int nx, int ny, int nz, double hx, double hy, double hz, const double *phi_dev,
                                  const double *x_dev, const double *y_dev, const double *z_dev, long long np, double ox, double oy,
                                  double oz, double *epx_dev, double *epy_dev, double *epz_dev, void *stream);

/* ---- One solve sharded over several GPUs (SURVEY.md sections 8(e), 8(f3)) ------------------------------------------------
 * The paper never splits a solve: several MPI ranks share ONE GPU through CUDA IPC.  This is the
 * contrasting B200 design: rank r of g (g a power of two <= 8; nx, ny, nz in [16, 256]) owns the y rows
 * [r ny/g, (r+1) ny/g) of rho and phi and the half-spectrum planes kz in [r nz/g, (r+1) nz/g) (the last rank also plane
 * nz).  P1 runs on the y slab and stores every output row directly into the receive buffer of the rank that owns its
 * plane; P2, P3, P4 run on the kz slab and P4 stores every row into the receive buffer of the rank that owns its y row;
 * P5 runs on the y slab.  The receive buffers are device pointers the caller makes peer-accessible (NVLink P2P /
 * symmetric memory; plain local pointers when several ranks are emulated on one device), so both exchanges -- two
 * all-to-alls of buffer A, 2 x 269 MB at 256^3 -- are the epilogues of the producing kernels, not separate collectives.
 * Between the phases the caller runs its own inter-rank barrier (e.g. an NCCL barrier on the same stream).
 *
 *   dks_poisson_set_shard     before the workspace is attached; changes dks_poisson_workspace_bytes(); afterwards
 *                             dks_poisson_set_max_batch (> 1) and dks_poisson_set_slab_planes are refused
 *   dks_greens_setup          every rank builds the full Green's octant (it only reads its own planes)
 *   dks_poisson_shard_buffers this rank's two receive buffers (inside its workspace), to be published to the peers
 *   dks_poisson_set_peers     tables of all ranks' receive buffers as seen from this device (entry `rank` = its own);
 *                             each table must hold nranks entries (the library reads exactly that many)
 *   dks_poisson_solve_shard   phase 1 (P1), barrier, phase 2 (P2-P4), barrier, phase 3 (P5); rho_loc / phi_loc are this
 *                             rank's y slabs, [nz][ny/g][nx] contiguous fp64 (rho_loc for phase 1, phi_loc for phase 3)
 * A sharded plan refuses dks_poisson_solve. */
int dks_poisson_set_shard(dks_poisson_plan *plan, int rank, int nranks);
int dks_poisson_shard_buffers(dks_poisson_plan *plan, void **recv_p1_dev, void **recv_p4_dev);
int dks_poisson_set_peers(dks_poisson_plan *plan, void *const *recv_p1_of_rank, void *const *recv_p4_of_rank);
int dks_poisson_solve_shard(dks_poisson_plan *plan, int phase, const double *rho_loc_dev, double *phi_loc_dev, void *stream);

/* Thread-local, NUL-terminated message describing the last failure in this thread ("" if none).  The library never
 * throws or aborts: every entry point reports through its status (the paper's DKS layer hands device errors back to
 * the host application in the same way). */
const char *dks_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* DKS_POISSON_H */

// dks_poisson.cu -- plan / workspace / stream management and the C ABI (include/dks_poisson.h).
//
// The plan owns: host metadata, device twiddle tables, profiling events, an ordering event between
// dks_greens_setup and dks_poisson_solve, and (unless the caller attached one) the device workspace
//     [ A | Ghat octant | host-path staging | B ].
// dks_poisson_solve launches five kernels on the caller's stream and returns; it neither allocates
// nor synchronises ("streams for asynchronous copy/compute").
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <mutex>
#include <new>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/dks_poisson.h"
#include "dks_passes_generic.cuh"
#include "dks_passes_r16.cuh"
#include "dks_passes_big.cuh"
#include "dks_greens_r16.cuh"
#include "dks_field_ops.cuh"

#ifndef DKS_PDL_MAX_NODES
#define DKS_PDL_MAX_NODES (1 << 21)   // programmatic dependent launch for meshes of at most this many nodes
#endif

using namespace dks;

// ------------------------------------------------------------------------------------------------
// errors
// ------------------------------------------------------------------------------------------------
static thread_local char g_err[512] = "";

static int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define DKS_CUDA(call)                                                                            \
    do {                                                                                          \
        cudaError_t e_ = (call);                                                                  \
        if (e_ != cudaSuccess)                                                                    \
            return fail(DKS_ERR_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_),     \
                        __FILE__, __LINE__);                                                      \
    } while (0)

extern "C" const char *dks_last_error(void) { return g_err; }

// ------------------------------------------------------------------------------------------------
// plan
// ------------------------------------------------------------------------------------------------
// Staging meshes of the host path.  A slot is busy from the start of its copy-in to the end of its copy-out (the solve runs in place
// on it): about 2.7 + 0.7 + 2.7 ms at 256^3 with both link directions busy.  Two slots allow one step per 3.05 ms; three make the
// pipeline link-bound (one step per copy time, 2.7 ms).
static const int kHostSlots = 3;

struct dks_poisson_plan {
    MeshDims d;
    double hx, hy, hz;
    double g0_override;                 // NaN = default rule
    // device
    int device = -1;
    int sm_count = 148;
    bool device_checked = false;
    cplx *tw[3] = { nullptr, nullptr, nullptr };   // twiddle tables for 2nx, 2ny, 2nz (may alias)
    std::vector<cplx> tw_host[3];
    // specialised (register-resident) passes: A = n / 16 per axis (0 = axis not supported), and the
    // between-step twiddle tables tw1[k A + a] = exp(-2 pi i a k / n), k < 16, a < A
    int r16A[3] = { 0, 0, 0 };
    cplx *tw1[3] = { nullptr, nullptr, nullptr };
    std::vector<cplx> tw1_host[3];
    bool fast[5] = { false, false, false, false, false };   // pass P1..P5 uses the r16 kernel
    int big[5] = { 0, 0, 0, 0, 0 };     // pass P1..P5 uses the long-line kernel with this padded length (1024 / 2048), else 0
    int bigL[3] = { 0, 0, 0 };          // per axis: 2n if n = 512 or 1024
    void *ws = nullptr;                 // workspace base
    size_t ws_bytes = 0;
    bool ws_owned = false;
    cplx *A = nullptr, *B = nullptr;
    double *G = nullptr, *stage = nullptr;   // stage: kHostSlots staging meshes (host path), back to back
    // host path pipeline (dks_poisson_solve_host_async): copy-in and copy-out streams and per-slot events
    cudaStream_t s_in = nullptr, s_out = nullptr;
    cudaEvent_t ev_in[kHostSlots] = {}, ev_solve[kHostSlots] = {}, ev_out[kHostSlots] = {};
    unsigned long long host_calls = 0;
    bool host_staging = true;           // the workspace carries the kHostSlots staging meshes (dks_poisson_set_host_staging; never on sharded plans)
    size_t offA, offB, offG, offS, need_bytes;
    // P2..P4 run slab by slab (slab = `slab` consecutive kz planes) so that B, the largest intermediate,
    // is a slab-sized scratch that stays resident in L2 between the three passes
    int slab = 0;                       // planes per slab, 1..nz+1
    bool slab_user = false;             // set through dks_poisson_set_slab_planes
    struct Step { int pass, kz0, planes; };     // pass 1..5
    // sharded solve (dks_poisson_set_shard): this plan is rank `rank` of `nranks`; it owns y rows [y0, y0 + ny_loc) of rho / phi
    // and half-spectrum planes [kz0, kz0 + planes_loc).  A1 = receive buffer of P1's rows [planes_loc][ny][nx] (it replaces A),
    // A2 = receive buffer of P4's rows [nz+1][ny_loc][nx].
    int rank = 0, nranks = 1, ny_loc = 0, y0 = 0, kz0 = 0, planes_loc = 0;
    cplx *A2 = nullptr;
    size_t offA2 = 0;
    PeerTable peers1 = PeerTable(), peers2 = PeerTable();
    bool peers_set = false;
    int max_batch = 1;                  // meshes per dks_poisson_solve_batch call the workspace is sized for
    bool pdl = false;                   // programmatic dependent launch between the r16 passes (small meshes)
    std::vector<Step> steps;            // the launch list of one solve
    bool greens_ready = false;
    bool setup_pending = false;         // setup_done not yet known to have completed
    cudaStream_t setup_stream = nullptr;   // stream dks_greens_setup launches on (dks_poisson_set_stream)
    cudaStream_t setup_used = nullptr;     // stream the current Ghat was built on
    cudaStream_t s_setup = nullptr;        // plan-owned stream of dks_poisson_step_host_async's rebuild
    cudaEvent_t setup_done = nullptr;
    cudaEvent_t ghat_free = nullptr;    // recorded after the last P3 of a solve that runs on another stream than the setup:
    bool ghat_free_recorded = false;    // the next rebuild of Ghat waits for it
    bool ghat_read_on_setup_stream = false;   // a solve ran on setup_used since the last rebuild: no event was recorded for it (stream
                                              // order covers a rebuild on that stream); a rebuild that moves to another stream records one then
    // profiling
    int prof_slots = 0;                 // 0 = off; else per-pass events of the last prof_slots solves are kept
    long long prof_count = 0;           // profiled solves issued since profiling was switched on
    std::vector<cudaEvent_t> ev;        // prof_slots * (kNumPasses + 1) events
    // generic-kernel launch parameters
    int Wx, Wy, Wz;                     // tile widths for lines along x / y / z
    size_t smem_x, smem_y, smem_z;
};

static const int kNumPasses = 5;
static const int kMaxProfSlots = 256;

static bool is_pow2_in_range(int n) { return n >= 8 && n <= 1024 && (n & (n - 1)) == 0; }
static int ilog2(int n) { int l = 0; while ((1 << l) < n) ++l; return l; }
static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

static int tile_width_for(int L)
{
    // shared memory per tile = L * (W+1) * 16 B; keep it <= ~80 KB so two or more CTAs fit per SM,
    // except for L = 2048 where W = 4 needs 160 KB.
    if (L <= 512) return 8;
    return 4;
}

// Bytes of B the L2 is asked to keep between P2, P3 and P4 of one slab (B200: 126 MB of L2).
static const size_t kSlabTargetBytes = (size_t)1 << 40;   // measured: slabbing loses, so automatic = one slab

static int auto_slab(const dks_poisson_plan *p)
{
    const size_t plane = (size_t)16 * p->d.nx * 2 * p->d.ny;
    const int planes = p->d.nz + 1;
    int s = (int)std::max<size_t>(1, kSlabTargetBytes / plane);
    if (s >= planes) return planes;
    const int count = (planes + s - 1) / s;          // equalise the slabs
    return (planes + count - 1) / count;
}

// [ A | Ghat | staging | B(slab) ]: B last, so that changing the slab size moves nothing else
static void compute_layout(dks_poisson_plan *p)
{
    const size_t nx = p->d.nx, ny = p->d.ny, nz = p->d.nz;
    size_t off = 0;
    const size_t nbm = (size_t)p->max_batch;
    if (p->nranks > 1) {                // A1 [planes_loc][ny][nx], A2 [nz+1][ny_loc][nx]
        p->offA = off; off = align_up(off + 16 * nx * ny * (size_t)p->planes_loc, 256);
        p->offA2 = off; off = align_up(off + 16 * nx * (size_t)p->ny_loc * (nz + 1), 256);
    } else {
        p->offA = off; off = align_up(off + 16 * nx * ny * (nz + 1) * nbm, 256);
    }
    p->offG = off; off = align_up(off + 8 * (size_t)p->d.gpitch * (ny + 1) * (nz + 1), 256);
    p->offS = off;
    if (p->host_staging && p->nranks == 1) off = align_up(off + kHostSlots * align_up(8 * nx * ny * nz, 256), 256);
    p->offB = off; off = align_up(off + 16 * nx * 2 * ny * (size_t)(p->nranks > 1 ? p->planes_loc : p->slab) * nbm, 256);
    p->need_bytes = off;
    p->steps.clear();
    p->steps.push_back({ 1, 0, 0 });
    for (int kz0 = 0; kz0 <= p->d.nz; kz0 += p->slab) {
        const int planes = std::min(p->slab, p->d.nz + 1 - kz0);
        p->steps.push_back({ 2, kz0, planes });
        p->steps.push_back({ 3, kz0, planes });
        p->steps.push_back({ 4, kz0, planes });
    }
    p->steps.push_back({ 5, 0, 0 });
}

static void bind_workspace(dks_poisson_plan *p)
{
    char *b = static_cast<char *>(p->ws);
    p->A = reinterpret_cast<cplx *>(b + p->offA);
    p->A2 = p->nranks > 1 ? reinterpret_cast<cplx *>(b + p->offA2) : nullptr;
    p->peers_set = false;
    p->B = reinterpret_cast<cplx *>(b + p->offB);
    p->G = reinterpret_cast<double *>(b + p->offG);
    p->stage = reinterpret_cast<double *>(b + p->offS);
}

extern "C" dks_poisson_plan *dks_poisson_plan_create(int nx, int ny, int nz, double hx, double hy, double hz)
{
    if (!is_pow2_in_range(nx) || !is_pow2_in_range(ny) || !is_pow2_in_range(nz)) {
        fail(DKS_ERR_INVALID_ARG, "mesh %dx%dx%d: every extent must be a power of two in [8, 1024]", nx, ny, nz);
        return nullptr;
    }
    if (!(hx > 0) || !(hy > 0) || !(hz > 0) || !std::isfinite(hx) || !std::isfinite(hy) || !std::isfinite(hz)) {
        fail(DKS_ERR_INVALID_ARG, "spacings must be finite and > 0 (got %g, %g, %g)", hx, hy, hz);
        return nullptr;
    }
    dks_poisson_plan *p = new (std::nothrow) dks_poisson_plan();
    if (!p) { fail(DKS_ERR_INVALID_ARG, "out of host memory"); return nullptr; }
    p->d.nx = nx; p->d.ny = ny; p->d.nz = nz;
    p->d.lx = ilog2(2 * nx); p->d.ly = ilog2(2 * ny); p->d.lz = ilog2(2 * nz);
    p->d.gpitch = (nx + 1 + 7) / 8 * 8;
    p->hx = hx; p->hy = hy; p->hz = hz;
    p->g0_override = std::nan("");
    const int Ls[3] = { 2 * nx, 2 * ny, 2 * nz };
    for (int a = 0; a < 3; ++a) {
        // tw[k] = exp(-2 pi i k / L), each entry straight from cosl/sinl with the argument reduced to
        // the first octant so that the table is exactly symmetric.
        const int L = Ls[a];
        p->tw_host[a].resize(L);
        const long double two_pi = 6.283185307179586476925286766559005768L;
        for (int k = 0; k < L; ++k) {
            long double th = two_pi * (long double)k / (long double)L;
            p->tw_host[a][k] = make_double2((double)cosl(th), (double)(-sinl(th)));
        }
    }
    const int ns[3] = { nx, ny, nz };
    for (int a = 0; a < 3; ++a) {
        const int n = ns[a];
        if (n < 16 || n > 256) continue;
        const int A = n / 16, L = 2 * n;
        p->r16A[a] = A;
        // three regions of n entries (dks_fft_r16.cuh, twiddle_between): exp(-2 pi i e / L) with
        //   e = 2 (t k mod n)                   parity 0
        //   e = 2 (t k mod n) + t               parity 1 forward:  w_n^(t k) w_L^t
        //   e = 2 (t k mod n) + (k mod A)       parity 1 inverse:  w_n^(t k) w_L^(k mod A)
        p->tw1_host[a].resize(3 * (size_t)n);
        const long double two_pi = 6.283185307179586476925286766559005768L;
        for (int region = 0; region < 3; ++region)
            for (int k = 0; k < 16; ++k)
                for (int t = 0; t < A; ++t) {
                    const int e = (2 * ((t * k) % n) + (region == 1 ? t : region == 2 ? k % A : 0)) % L;
                    long double th = two_pi * (long double)e / (long double)L;
                    p->tw1_host[a][(size_t)region * n + k * A + t] = make_double2((double)cosl(th), (double)(-sinl(th)));
                }
    }
    // P1/P5 run along z and need 16 real columns per CTA; P2/P4 along y; P3 along x (nx = 256 only)
    for (int a = 0; a < 3; ++a) p->bigL[a] = (ns[a] == 512 || ns[a] == 1024) ? 2 * ns[a] : 0;
    p->big[0] = p->big[4] = (p->bigL[2] && nx >= 2 * (p->bigL[2] == 1024 ? BigGeom<1024>::W : BigGeom<2048>::W)) ? p->bigL[2] : 0;
    p->big[1] = p->big[3] = p->bigL[1];
    p->big[2] = p->bigL[0];
    p->fast[0] = p->fast[4] = p->r16A[2] != 0 && nx >= 16;
    p->fast[1] = p->fast[3] = p->r16A[1] != 0;
    p->fast[2] = p->r16A[0] != 0;
    // tile widths: lines along x are tiled over ky (2ny >= 16 of them per plane); lines along y / z are
    // tiled over x (nx complex columns, or nx/2 packed real pairs for the z passes)
    p->Wx = tile_width_for(2 * nx);
    p->Wy = std::min(tile_width_for(2 * ny), nx);
    p->Wz = std::min(tile_width_for(2 * nz), nx / 2);
    p->smem_x = (size_t)2 * nx * (p->Wx + 1) * sizeof(cplx);
    p->smem_y = (size_t)2 * ny * p->Wy * sizeof(cplx);
    p->smem_z = (size_t)2 * nz * p->Wz * sizeof(cplx);
    p->slab = auto_slab(p);
    p->pdl = (size_t)nx * ny * nz <= (size_t)DKS_PDL_MAX_NODES;
    compute_layout(p);
    g_err[0] = 0;
    return p;
}

static void release_device(dks_poisson_plan *p)
{
    for (int a = 0; a < 3; ++a) {
        bool alias = false;
        for (int b = 0; b < a; ++b) alias |= (p->tw[b] == p->tw[a]);
        if (p->tw[a] && !alias) cudaFree(p->tw[a]);
    }
    for (int a = 0; a < 3; ++a) p->tw[a] = nullptr;
    for (int a = 0; a < 3; ++a) {
        if (p->tw1[a]) cudaFree(p->tw1[a]);     // never aliased
        p->tw1[a] = nullptr;
    }
    if (p->ws_owned && p->ws) cudaFree(p->ws);
    p->ws = nullptr; p->ws_owned = false;
    if (p->setup_done) cudaEventDestroy(p->setup_done);
    if (p->ghat_free) cudaEventDestroy(p->ghat_free);
    p->setup_done = p->ghat_free = nullptr;
    if (p->s_setup) cudaStreamDestroy(p->s_setup);
    p->s_setup = nullptr;
    for (int i = 0; i < kHostSlots; ++i) {
        if (p->ev_in[i]) cudaEventDestroy(p->ev_in[i]);
        if (p->ev_solve[i]) cudaEventDestroy(p->ev_solve[i]);
        if (p->ev_out[i]) cudaEventDestroy(p->ev_out[i]);
        p->ev_in[i] = p->ev_solve[i] = p->ev_out[i] = nullptr;
    }
    if (p->s_in) cudaStreamDestroy(p->s_in);
    if (p->s_out) cudaStreamDestroy(p->s_out);
    p->s_in = p->s_out = nullptr;
    for (auto &e : p->ev) if (e) cudaEventDestroy(e);
    p->ev.clear();
}

extern "C" void dks_poisson_plan_destroy(dks_poisson_plan *p)
{
    if (!p) return;
    release_device(p);
    delete p;
}

// ------------------------------------------------------------------------------------------------
// specialised passes: attribute setup and launch by A = n / 16
// ------------------------------------------------------------------------------------------------
#define DKS_FOR_EACH_A(X) X(1) X(2) X(4) X(8) X(16)

static int r16_set_attributes()
{
#define X(A_)                                                                                                         \
    DKS_CUDA(cudaFuncSetAttribute(p1_z_r2c_r16<A_, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, P1Geom<A_>::SMEM));  \
    DKS_CUDA(cudaFuncSetAttribute(p1_z_r2c_r16<A_, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, P1Geom<A_>::SMEM));  \
    DKS_CUDA(cudaFuncSetAttribute(p1_z_r2c_r16<A_, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, P1Geom<A_>::SMEM));  \
    DKS_CUDA(cudaFuncSetAttribute(p4_y_inv_r16<A_, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, R16Geom<A_>::SMEM)); \
    DKS_CUDA(cudaFuncSetAttribute(p2_y_fwd_r16<A_, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, R16Geom<A_>::SMEM)); \
    DKS_CUDA(cudaFuncSetAttribute(p2_y_fwd_r16<A_, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, R16Geom<A_>::SMEM)); \
    DKS_CUDA(cudaFuncSetAttribute(p1_z_r2c_r16p<A_, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, R16Geom<A_>::SMEM / 2)); \
    DKS_CUDA(cudaFuncSetAttribute(p1_z_r2c_r16p<A_, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, R16Geom<A_>::SMEM / 2)); \
    DKS_CUDA(cudaFuncSetAttribute(p2_y_fwd_r16p<A_, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, R16Geom<A_>::SMEM / 2)); \
    DKS_CUDA(cudaFuncSetAttribute(p2_y_fwd_r16p<A_, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, R16Geom<A_>::SMEM / 2)); \
    DKS_CUDA(cudaFuncSetAttribute(p4_y_inv_r16<A_, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, R16Geom<A_>::SMEM)); \
    DKS_CUDA(cudaFuncSetAttribute(p4_y_inv_r16<A_, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, R16Geom<A_>::SMEM)); \
    DKS_CUDA(cudaFuncSetAttribute(p5_z_c2r_r16<A_, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, R16Geom<A_>::SMEM)); \
    DKS_CUDA(cudaFuncSetAttribute(p5_z_c2r_r16<A_, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, R16Geom<A_>::SMEM)); \
    DKS_CUDA(cudaFuncSetAttribute(p3_x_conv_r16<A_, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kP3Smem)); \
    DKS_CUDA(cudaFuncSetAttribute(p3_x_conv_r16<A_, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kP3Smem)); \
    DKS_CUDA(cudaFuncSetAttribute(greens_x_r16<A_>, cudaFuncAttributeMaxDynamicSharedMemorySize, kGxSmem)); \
    DKS_CUDA(cudaFuncSetAttribute(greens_axis_r16<A_>, cudaFuncAttributeMaxDynamicSharedMemorySize, R16Geom<A_>::SMEM));
    DKS_FOR_EACH_A(X)
#undef X
    return DKS_OK;
}

// Launch with programmatic stream serialization (programmatic dependent launch): the kernel may be scheduled
// while the previous kernel in the stream drains; it orders itself with pdl_wait() (dks_common.cuh).
// Measured: it hides 2-3 us per kernel boundary on the small meshes (128^3: 0.113 -> 0.104 ms, 64^3: 0.037 -> 0.034 ms)
// but costs 5 % at 256^3, so the plan enables it for meshes of at most 128^3 nodes (`pdl`).
template <typename... KArgs, typename... Args>
static void launch_pdl(bool pdl, void (*kernel)(KArgs...), void (*kernel_pdl)(KArgs...), dim3 grid, dim3 block, size_t smem,
                       cudaStream_t st, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    if (!pdl) {
        kernel<<<grid, block, smem, st>>>(static_cast<KArgs>(args)...);
        return;
    }
    cfg.attrs = attr; cfg.numAttrs = 1;
    (void)cudaLaunchKernelEx(&cfg, kernel_pdl, static_cast<KArgs>(args)...);      // errors surface through cudaGetLastError in the solve
}

template <int A>
static void launch_strided_r16(const dks_poisson_plan::Step &s, const dks_poisson_plan *p, const double *rho, double *phi,
                               int nb, cudaStream_t st)
{
    const MeshDims d = p->d;
    const int T = R16Geom<A>::THREADS, S = R16Geom<A>::SMEM;
    switch (s.pass) {
    case 1: {
        if (A >= kSplitMinA) {                          // one CTA per parity (CTAs of at least two warps)
            launch_pdl(p->pdl, p1_z_r2c_r16p<A, false>, p1_z_r2c_r16p<A, true>, dim3(2 * d.nx / (2 * kCols), d.ny, nb), dim3(T / 2), S / 2, st, rho, p->A, d, p->tw1[2], p->tw[2]);
            break;
        }
        const int tiles = d.nx / (2 * kCols) * d.ny * nb, per_sm = std::max(1, std::min(512 / T, (227 * 1024) / (P1Geom<A>::SMEM + 1024)));
        launch_pdl(p->pdl, p1_z_r2c_r16<A, false>, p1_z_r2c_r16<A, true>, dim3(std::min(tiles, p->sm_count * per_sm)), dim3(T), P1Geom<A>::SMEM, st, rho, p->A, d, nb, p->tw1[2], p->tw[2], PeerTable());
        break;
    }
    case 2:
        if (A >= kSplitMinA)
            launch_pdl(p->pdl, p2_y_fwd_r16p<A, false>, p2_y_fwd_r16p<A, true>, dim3(2 * d.nx / kCols, s.planes * nb), dim3(T / 2), S / 2, st, p->A, p->B, d, s.kz0, p->tw1[1], p->tw[1]);
        else
            launch_pdl(p->pdl, p2_y_fwd_r16<A, false>, p2_y_fwd_r16<A, true>, dim3(d.nx / kCols, s.planes * nb), dim3(T), S, st, p->A, p->B, d, s.kz0, p->tw1[1], p->tw[1]);
        break;
    case 4: launch_pdl(p->pdl, p4_y_inv_r16<A, false>, p4_y_inv_r16<A, true>, dim3(d.nx / kCols, s.planes * nb), dim3(T), S, st, p->B, p->A, d, s.kz0, p->tw1[1], p->tw[1], PeerTable()); break;
    case 5: launch_pdl(p->pdl, p5_z_c2r_r16<A, false>, p5_z_c2r_r16<A, true>, dim3(d.nx / (2 * kCols), d.ny, nb), dim3(T), S, st, p->A, phi, d, p->tw1[2], p->tw[2]); break;
    }
}

static void launch_r16(const dks_poisson_plan::Step &s, const dks_poisson_plan *p, const double *rho, double *phi,
                       int nb, cudaStream_t st)
{
    if (s.pass == 3) {
        const MeshDims d = p->d;
        const unsigned groups = (unsigned)s.planes * nb * 2 * d.ny / (16 / p->r16A[0]);      // 256 complex each
        const unsigned grid = std::min<unsigned>((unsigned)p->sm_count, (groups + kP3Warps - 1) / kP3Warps);
        switch (p->r16A[0]) {
#define X(A_) case A_: launch_pdl(p->pdl, p3_x_conv_r16<A_, false>, p3_x_conv_r16<A_, true>, dim3(grid), dim3(kP3Warps * 32), kP3Smem, st, p->B, p->G, d, s.kz0, s.planes * nb, p->tw1[0]); break;
            DKS_FOR_EACH_A(X)
#undef X
        }
        return;
    }
    const int A = (s.pass == 1 || s.pass == 5) ? p->r16A[2] : p->r16A[1];
    switch (A) {
#define X(A_) case A_: launch_strided_r16<A_>(s, p, rho, phi, nb, st); break;
        DKS_FOR_EACH_A(X)
#undef X
    }
}

template <int L>
static void launch_big(const dks_poisson_plan::Step &s, const dks_poisson_plan *p, const double *rho, double *phi,
                       int nb, cudaStream_t st)
{
    typedef BigGeom<L> G;
    const MeshDims d = p->d;
    switch (s.pass) {
    case 1: launch_pdl(p->pdl, p1_z_r2c_big<L, false>, p1_z_r2c_big<L, true>, dim3(d.nx / (2 * G::W), d.ny, nb), dim3(G::THREADS), G::SMEM, st, rho, p->A, d, p->tw[2]); break;
    case 2: launch_pdl(p->pdl, p2_y_fwd_big<L, false>, p2_y_fwd_big<L, true>, dim3(d.nx / G::W, s.planes * nb), dim3(G::THREADS), G::SMEM, st, p->A, p->B, d, s.kz0, p->tw[1]); break;
    case 3: launch_pdl(p->pdl, p3_x_conv_big<L, false>, p3_x_conv_big<L, true>, dim3((unsigned)((size_t)s.planes * nb * 2 * d.ny / P3BigGeom<L>::W)), dim3(P3BigGeom<L>::THREADS), P3BigGeom<L>::SMEM, st, p->B, p->G, d, s.kz0, p->tw[0]); break;
    case 4: launch_pdl(p->pdl, p4_y_inv_big<L, false>, p4_y_inv_big<L, true>, dim3(d.nx / G::W, s.planes * nb), dim3(G::THREADS), G::SMEM, st, p->B, p->A, d, s.kz0, p->tw[1]); break;
    case 5: launch_pdl(p->pdl, p5_z_c2r_big<L, false>, p5_z_c2r_big<L, true>, dim3(d.nx / (2 * G::W), d.ny, nb), dim3(G::THREADS), G::SMEM, st, p->A, phi, d, p->tw[2]); break;
    }
}

template <int L>
static int big_set_attributes()
{
    typedef BigGeom<L> G;
    DKS_CUDA(cudaFuncSetAttribute(p1_z_r2c_big<L, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, G::SMEM));
    DKS_CUDA(cudaFuncSetAttribute(p1_z_r2c_big<L, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, G::SMEM));
    DKS_CUDA(cudaFuncSetAttribute(p2_y_fwd_big<L, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, G::SMEM));
    DKS_CUDA(cudaFuncSetAttribute(p2_y_fwd_big<L, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, G::SMEM));
    DKS_CUDA(cudaFuncSetAttribute(p3_x_conv_big<L, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, P3BigGeom<L>::SMEM));
    DKS_CUDA(cudaFuncSetAttribute(p3_x_conv_big<L, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, P3BigGeom<L>::SMEM));
    DKS_CUDA(cudaFuncSetAttribute(p4_y_inv_big<L, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, G::SMEM));
    DKS_CUDA(cudaFuncSetAttribute(p4_y_inv_big<L, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, G::SMEM));
    DKS_CUDA(cudaFuncSetAttribute(p5_z_c2r_big<L, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, G::SMEM));
    DKS_CUDA(cudaFuncSetAttribute(p5_z_c2r_big<L, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, G::SMEM));
    DKS_CUDA(cudaFuncSetAttribute(greens_axis_big<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, G::SMEMX));
    return DKS_OK;
}

static void launch_generic(const dks_poisson_plan::Step &s, const dks_poisson_plan *p, const double *rho, double *phi,
                           int nb, cudaStream_t st)
{
    const MeshDims d = p->d;
    switch (s.pass) {
    case 1: p1_z_r2c_generic<<<dim3(d.nx / (2 * p->Wz), d.ny, nb), 256, p->smem_z, st>>>(rho, p->A, d, p->Wz, p->tw[2]); break;
    case 2: p2_y_fwd_generic<<<dim3(d.nx / p->Wy, s.planes * nb), 256, p->smem_y, st>>>(p->A, p->B, d, s.kz0, p->Wy, p->tw[1]); break;
    case 3: p3_x_conv_generic<<<(unsigned)((size_t)s.planes * nb * 2 * d.ny / p->Wx), 256, p->smem_x, st>>>(p->B, p->G, d, s.kz0,
                                                                                                    p->Wx, p->tw[0]); break;
    case 4: p4_y_inv_generic<<<dim3(d.nx / p->Wy, s.planes * nb), 256, p->smem_y, st>>>(p->B, p->A, d, s.kz0, p->Wy, p->tw[1]); break;
    case 5: p5_z_c2r_generic<<<dim3(d.nx / (2 * p->Wz), d.ny, nb), 256, p->smem_z, st>>>(p->A, phi, d, p->Wz, p->tw[2]); break;
    }
}

// First device touch: check the architecture, upload twiddles, create events, opt in to large smem.
static int ensure_device(dks_poisson_plan *p)
{
    if (p->device_checked) return DKS_OK;
    int dev = 0;
    DKS_CUDA(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    DKS_CUDA(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10)
        return fail(DKS_ERR_UNSUPPORTED_DEVICE, "device %d (%s) is compute capability %d.%d; this library is built for sm_100a only",
                    dev, prop.name, prop.major, prop.minor);
    p->device = dev;
    p->sm_count = prop.multiProcessorCount;
    const int Ls[3] = { 2 * p->d.nx, 2 * p->d.ny, 2 * p->d.nz };
    for (int a = 0; a < 3; ++a) {
        for (int b = 0; b < a; ++b) if (Ls[b] == Ls[a]) p->tw[a] = p->tw[b];
        if (p->tw[a]) continue;
        DKS_CUDA(cudaMalloc(&p->tw[a], sizeof(cplx) * Ls[a]));
        DKS_CUDA(cudaMemcpy(p->tw[a], p->tw_host[a].data(), sizeof(cplx) * Ls[a], cudaMemcpyHostToDevice));
    }
    for (int a = 0; a < 3; ++a) {
        if (!p->r16A[a] || p->tw1[a]) continue;
        const size_t bytes = sizeof(cplx) * p->tw1_host[a].size();
        DKS_CUDA(cudaMalloc(&p->tw1[a], bytes));
        DKS_CUDA(cudaMemcpy(p->tw1[a], p->tw1_host[a].data(), bytes, cudaMemcpyHostToDevice));
    }
    DKS_CUDA(cudaEventCreateWithFlags(&p->setup_done, cudaEventDisableTiming));
    // cudaFuncAttributeMaxDynamicSharedMemorySize is a setter, not a running maximum, and the kernels are shared by all
    // plans of the process: set every kernel once per device to the largest size any supported mesh needs (n = 1024).
    static bool attributes_set[64] = {};
    if (dev >= 64 || !attributes_set[dev]) {
        const int kMaxL = 2048;
        const size_t smem_strided = (size_t)kMaxL * tile_width_for(kMaxL) * sizeof(cplx);            // lines along y / z
        const size_t smem_lines = (size_t)kMaxL * (tile_width_for(kMaxL) + 1) * sizeof(cplx);        // lines along x, Green's axes
        if ((size_t)prop.sharedMemPerBlockOptin < smem_lines)
            return fail(DKS_ERR_UNSUPPORTED_DEVICE, "device offers %zu B of shared memory per block, %zu needed",
                        (size_t)prop.sharedMemPerBlockOptin, smem_lines);
        DKS_CUDA(cudaFuncSetAttribute(p1_z_r2c_generic, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_strided));
        DKS_CUDA(cudaFuncSetAttribute(p5_z_c2r_generic, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_strided));
        DKS_CUDA(cudaFuncSetAttribute(p2_y_fwd_generic, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_strided));
        DKS_CUDA(cudaFuncSetAttribute(p4_y_inv_generic, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_strided));
        DKS_CUDA(cudaFuncSetAttribute(p3_x_conv_generic, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_lines));
        DKS_CUDA(cudaFuncSetAttribute(greens_axis_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_lines));
        int rc = r16_set_attributes();
        if (rc) return rc;
        if ((rc = big_set_attributes<1024>()) || (rc = big_set_attributes<2048>())) return rc;
        if (dev < 64) attributes_set[dev] = true;
    }
    DKS_CUDA(cudaEventCreateWithFlags(&p->ghat_free, cudaEventDisableTiming));
    p->device_checked = true;
    return DKS_OK;
}

extern "C" size_t dks_poisson_workspace_bytes(const dks_poisson_plan *p)
{
    if (!p) { fail(DKS_ERR_INVALID_ARG, "plan is NULL"); return 0; }
    return p->need_bytes;
}

extern "C" int dks_poisson_set_workspace(dks_poisson_plan *p, void *dev_ptr, size_t bytes)
{
    if (!p || !dev_ptr) return fail(DKS_ERR_INVALID_ARG, "plan or workspace pointer is NULL");
    if (reinterpret_cast<uintptr_t>(dev_ptr) % 256) return fail(DKS_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
    if (bytes < p->need_bytes)
        return fail(DKS_ERR_WORKSPACE_TOO_SMALL, "workspace has %zu bytes, %zu needed", bytes, p->need_bytes);
    if (p->ws_owned && p->ws) cudaFree(p->ws);
    p->ws = dev_ptr; p->ws_bytes = bytes; p->ws_owned = false;
    bind_workspace(p);
    p->greens_ready = false;
    return DKS_OK;
}

extern "C" int dks_poisson_set_slab_planes(dks_poisson_plan *p, int planes)
{
    if (!p) return fail(DKS_ERR_INVALID_ARG, "plan is NULL");
    if (planes < 0 || planes > p->d.nz + 1) return fail(DKS_ERR_INVALID_ARG, "planes must be in [0, nz+1] (0 = automatic)");
    if (p->nranks > 1) return fail(DKS_ERR_INVALID_ARG, "sharding excludes slabs (this plan is rank %d of %d)", p->rank, p->nranks);
    const int old = p->slab;
    p->slab = planes ? planes : auto_slab(p);
    compute_layout(p);
    if (p->ws && p->ws_bytes < p->need_bytes) {
        const size_t need = p->need_bytes;
        p->slab = old;
        compute_layout(p);
        return fail(DKS_ERR_WORKSPACE_TOO_SMALL, "the attached workspace has %zu bytes, %zu needed for slabs of %d planes; "
                    "set the slab size before attaching the workspace / before dks_greens_setup", p->ws_bytes, need, planes);
    }
    p->slab_user = planes != 0;
    p->prof_slots = 0;                  // the launch list changed: recorded events no longer match
    if (p->ws) bind_workspace(p);
    return DKS_OK;
}

extern "C" int dks_poisson_slab_planes(const dks_poisson_plan *p)
{
    if (!p) return fail(DKS_ERR_INVALID_ARG, "plan is NULL");
    return p->slab;
}

extern "C" int dks_poisson_set_stream(dks_poisson_plan *p, void *stream)
{
    if (!p) return fail(DKS_ERR_INVALID_ARG, "plan is NULL");
    p->setup_stream = static_cast<cudaStream_t>(stream);
    return DKS_OK;
}

extern "C" int dks_poisson_set_spacing(dks_poisson_plan *p, double hx, double hy, double hz)
{
    if (!p) return fail(DKS_ERR_INVALID_ARG, "plan is NULL");
    if (!(hx > 0) || !(hy > 0) || !(hz > 0) || !std::isfinite(hx) || !std::isfinite(hy) || !std::isfinite(hz))
        return fail(DKS_ERR_INVALID_ARG, "spacings must be finite and > 0 (got %g, %g, %g)", hx, hy, hz);
    p->hx = hx; p->hy = hy; p->hz = hz;
    p->greens_ready = false;
    return DKS_OK;
}

extern "C" int dks_poisson_set_g0(dks_poisson_plan *p, double g0)
{
    if (!p) return fail(DKS_ERR_INVALID_ARG, "plan is NULL");
    if (std::isinf(g0)) return fail(DKS_ERR_INVALID_ARG, "g0 must be finite or NaN");
    p->g0_override = g0;
    p->greens_ready = false;
    return DKS_OK;
}

// ------------------------------------------------------------------------------------------------
// a0: Green's function build + transform
// ------------------------------------------------------------------------------------------------
static int greens_setup_on(dks_poisson_plan *p, cudaStream_t st)
{
    int rc = ensure_device(p);
    if (rc) return rc;
    if (!p->ws) {
        DKS_CUDA(cudaMalloc(&p->ws, p->need_bytes));
        p->ws_bytes = p->need_bytes; p->ws_owned = true;
        bind_workspace(p);
    }
    const MeshDims d = p->d;
    // The rebuild overwrites Ghat in place, in three passes.  Order it after (1) the last P3 issued on another stream (P3 is the
    // only reader of Ghat), (2) a previous build still running on another stream, (3) solves that ran on the previous build's own
    // stream: those record no event per solve (it would sit between P3 and P4 of every solve), so one is recorded now, at the
    // current tail of that stream -- behind the whole solve, which is more than needed but happens once per change of stream.
    if (p->ghat_free_recorded) DKS_CUDA(cudaStreamWaitEvent(st, p->ghat_free, 0));
    if (st != p->setup_used) {
        if (p->setup_pending) DKS_CUDA(cudaStreamWaitEvent(st, p->setup_done, 0));
        if (p->ghat_read_on_setup_stream) {
            DKS_CUDA(cudaEventRecord(p->ghat_free, p->setup_used));
            DKS_CUDA(cudaStreamWaitEvent(st, p->ghat_free, 0));
            p->ghat_free_recorded = true;
        }
    }
    p->ghat_read_on_setup_stream = false;
    // 1/(4 pi eps0), eps0 = 8.8541878128e-12 F/m (CODATA 2018), evaluated in long double.
    const long double pi_l = 3.141592653589793238462643383279502884L;
    const double coef = (double)(1.0L / (4.0L * pi_l * 8.8541878128e-12L));
    const double hmin = std::min(p->hx, std::min(p->hy, p->hz));
    const double g0 = std::isnan(p->g0_override) ? coef / (0.5 * hmin) : p->g0_override;
    const long long pitch = d.gpitch, plane = pitch * (d.ny + 1);
    const int W = 4;
    // fold hx hy hz / (8 nx ny nz) (Eq. (2)'s prefactor and the inverse transform's 1/N, reading A5) into the last axis
    const double scale = p->hx * p->hy * p->hz / (8.0 * d.nx * d.ny * d.nz);
    // x lines: (ky, kz) ; y lines: (kx, kz) ; z lines: (kx, ky).  Every axis with n = 32..256 takes the
    // register-resident kernels of dks_greens_r16.cuh (x: fused with the evaluation of G), the others the generic ones.
    if (p->r16A[0]) {
        const unsigned pairs = (unsigned)(d.nz + 1) * ((d.ny + 2) / 2), groups = (pairs + 16 / p->r16A[0] - 1) / (16 / p->r16A[0]);
        const unsigned grid = std::min<unsigned>((unsigned)p->sm_count, (groups + kGxWarps - 1) / kGxWarps);
        switch (p->r16A[0]) {
#define X(A_) case A_: greens_x_r16<A_><<<grid, kGxWarps * 32, kGxSmem, st>>>(p->G, d, p->hx, p->hy, p->hz, coef, g0, p->tw1[0]); break;
            DKS_FOR_EACH_A(X)
#undef X
        }
    } else {
        dim3 blk(128), grd((d.gpitch + 127) / 128, d.ny + 1, d.nz + 1);
        greens_fill_kernel<<<grd, blk, 0, st>>>(p->G, d, p->hx, p->hy, p->hz, coef, g0);
        long long nl = (long long)(d.ny + 1) * (d.nz + 1);
        size_t sm = (size_t)2 * d.nx * (W + 1) * sizeof(cplx);
        if (p->bigL[0] == 1024) greens_axis_big<1024><<<(unsigned)((nl + 2 * BigGeom<1024>::W - 1) / (2 * BigGeom<1024>::W)), BigGeom<1024>::THREADS, BigGeom<1024>::SMEMX, st>>>(p->G, 1, d.ny + 1, pitch, d.nz + 1, plane, 1.0, p->tw[0]);
        else if (p->bigL[0] == 2048) greens_axis_big<2048><<<(unsigned)((nl + 2 * BigGeom<2048>::W - 1) / (2 * BigGeom<2048>::W)), BigGeom<2048>::THREADS, BigGeom<2048>::SMEMX, st>>>(p->G, 1, d.ny + 1, pitch, d.nz + 1, plane, 1.0, p->tw[0]);
        else
        greens_axis_kernel<<<(unsigned)((nl + 2 * W - 1) / (2 * W)), 256, sm, st>>>(p->G, d.nx, d.lx, W, 1, d.ny + 1, pitch,
                                                                                   d.nz + 1, plane, 1.0, p->tw[0]);
    }
    const dim3 xt((d.gpitch + 2 * kCols - 1) / (2 * kCols));
    if (p->r16A[1]) {
        switch (p->r16A[1]) {
#define X(A_) case A_: greens_axis_r16<A_><<<dim3(xt.x, d.nz + 1), R16Geom<A_>::THREADS, R16Geom<A_>::SMEM, st>>>(p->G, d.gpitch, pitch, plane, 1.0, p->tw1[1]); break;
            DKS_FOR_EACH_A(X)
#undef X
        }
    } else {
        long long nl = (long long)(d.nx + 1) * (d.nz + 1);
        size_t sm = (size_t)2 * d.ny * (W + 1) * sizeof(cplx);
        if (p->bigL[1] == 1024) greens_axis_big<1024><<<(unsigned)((nl + 2 * BigGeom<1024>::W - 1) / (2 * BigGeom<1024>::W)), BigGeom<1024>::THREADS, BigGeom<1024>::SMEMX, st>>>(p->G, pitch, d.nx + 1, 1, d.nz + 1, plane, 1.0, p->tw[1]);
        else if (p->bigL[1] == 2048) greens_axis_big<2048><<<(unsigned)((nl + 2 * BigGeom<2048>::W - 1) / (2 * BigGeom<2048>::W)), BigGeom<2048>::THREADS, BigGeom<2048>::SMEMX, st>>>(p->G, pitch, d.nx + 1, 1, d.nz + 1, plane, 1.0, p->tw[1]);
        else
        greens_axis_kernel<<<(unsigned)((nl + 2 * W - 1) / (2 * W)), 256, sm, st>>>(p->G, d.ny, d.ly, W, pitch, d.nx + 1, 1,
                                                                                   d.nz + 1, plane, 1.0, p->tw[1]);
    }
    if (p->r16A[2]) {
        switch (p->r16A[2]) {
#define X(A_) case A_: greens_axis_r16<A_><<<dim3(xt.x, d.ny + 1), R16Geom<A_>::THREADS, R16Geom<A_>::SMEM, st>>>(p->G, d.gpitch, plane, pitch, scale, p->tw1[2]); break;
            DKS_FOR_EACH_A(X)
#undef X
        }
    } else {
        long long nl = (long long)(d.nx + 1) * (d.ny + 1);
        size_t sm = (size_t)2 * d.nz * (W + 1) * sizeof(cplx);
        if (p->bigL[2] == 1024) greens_axis_big<1024><<<(unsigned)((nl + 2 * BigGeom<1024>::W - 1) / (2 * BigGeom<1024>::W)), BigGeom<1024>::THREADS, BigGeom<1024>::SMEMX, st>>>(p->G, plane, d.nx + 1, 1, d.ny + 1, pitch, scale, p->tw[2]);
        else if (p->bigL[2] == 2048) greens_axis_big<2048><<<(unsigned)((nl + 2 * BigGeom<2048>::W - 1) / (2 * BigGeom<2048>::W)), BigGeom<2048>::THREADS, BigGeom<2048>::SMEMX, st>>>(p->G, plane, d.nx + 1, 1, d.ny + 1, pitch, scale, p->tw[2]);
        else
        greens_axis_kernel<<<(unsigned)((nl + 2 * W - 1) / (2 * W)), 256, sm, st>>>(p->G, d.nz, d.lz, W, plane, d.nx + 1, 1,
                                                                                   d.ny + 1, pitch, scale, p->tw[2]);
    }
    DKS_CUDA(cudaGetLastError());
    DKS_CUDA(cudaEventRecord(p->setup_done, st));
    p->greens_ready = true;
    p->setup_pending = true;
    p->setup_used = st;
    return DKS_OK;
}

extern "C" int dks_greens_setup(dks_poisson_plan *p)
{
    if (!p) return fail(DKS_ERR_INVALID_ARG, "plan is NULL");
    return greens_setup_on(p, p->setup_stream);
}

extern "C" int dks_poisson_copy_greens_hat(dks_poisson_plan *p, double *host_out)
{
    if (!p || !host_out) return fail(DKS_ERR_INVALID_ARG, "plan or output pointer is NULL");
    if (!p->greens_ready) return fail(DKS_ERR_NOT_SETUP, "dks_greens_setup has not been called");
    DKS_CUDA(cudaEventSynchronize(p->setup_done));
    const MeshDims d = p->d;
    DKS_CUDA(cudaMemcpy2D(host_out, sizeof(double) * (d.nx + 1), p->G, sizeof(double) * d.gpitch,
                          sizeof(double) * (d.nx + 1), (size_t)(d.ny + 1) * (d.nz + 1), cudaMemcpyDeviceToHost));
    return DKS_OK;
}

// ------------------------------------------------------------------------------------------------
// the solve
// ------------------------------------------------------------------------------------------------
extern "C" int dks_poisson_launches_per_solve(const dks_poisson_plan *p)
{
    if (!p) return fail(DKS_ERR_INVALID_ARG, "plan is NULL");
    return (int)p->steps.size();
}

extern "C" double dks_poisson_model_bytes(const dks_poisson_plan *p, int pass)
{
    if (!p) { fail(DKS_ERR_INVALID_ARG, "plan is NULL"); return 0.0; }
    const double nx = p->d.nx, ny = p->d.ny, nz = p->d.nz;
    const double rho = 8 * nx * ny * nz, a = 16 * nx * ny * (nz + 1), b = 2 * a;
    const double g = 8 * (nx + 1) * (ny + 1) * (nz + 1);
    switch (pass) {
    case 0: return 2 * rho + 4 * a + 4 * b + g;
    case 1: return rho + a;
    case 2: return a + b;
    case 3: return 2 * b + g;
    case 4: return a + b;
    case 5: return rho + a;
    default: fail(DKS_ERR_INVALID_ARG, "pass must be 0..5"); return 0.0;
    }
}

extern "C" const char *dks_poisson_pass_name(const dks_poisson_plan *p, int pass)
{
    if (!p || pass < 1 || pass > 5) { fail(DKS_ERR_INVALID_ARG, "bad plan or pass"); return ""; }
    static const char *names[5] = { "p1_z_r2c_generic", "p2_y_fwd_generic", "p3_x_conv_generic",
                                    "p4_y_inv_generic", "p5_z_c2r_generic" };
    static const char *fast_names[5] = { "p1_z_r2c_r16", "p2_y_fwd_r16", "p3_x_conv_r16", "p4_y_inv_r16", "p5_z_c2r_r16" };
    static const char *big_names[5] = { "p1_z_r2c_big", "p2_y_fwd_big", "p3_x_conv_big", "p4_y_inv_big", "p5_z_c2r_big" };
    // P1 and P2 run one CTA per parity where a parity's CTA has at least two warps (launch_strided_r16)
    if (pass == 1 && p->fast[0] && p->r16A[2] >= kSplitMinA && p->nranks == 1) return "p1_z_r2c_r16p";
    if (pass == 2 && p->fast[1] && p->r16A[1] >= kSplitMinA) return "p2_y_fwd_r16p";
    return p->fast[pass - 1] ? fast_names[pass - 1] : p->big[pass - 1] ? big_names[pass - 1] : names[pass - 1];
}

// Events of one profiled solve: one before every launch of the launch list and one after the last.
static size_t prof_stride(const dks_poisson_plan *p) { return p->steps.size() + 1; }

extern "C" int dks_poisson_set_profiling(dks_poisson_plan *p, int slots)
{
    if (!p) return fail(DKS_ERR_INVALID_ARG, "plan is NULL");
    if (slots < 0 || slots > kMaxProfSlots) return fail(DKS_ERR_INVALID_ARG, "slots must be in [0, %d]", kMaxProfSlots);
    if (slots > 0) {
        int rc = ensure_device(p);
        if (rc) return rc;
    }
    const size_t need = (size_t)slots * prof_stride(p);
    while (p->ev.size() < need) {
        cudaEvent_t e;
        DKS_CUDA(cudaEventCreate(&e));
        p->ev.push_back(e);
    }
    p->prof_slots = slots;
    p->prof_count = 0;
    return DKS_OK;
}

extern "C" int dks_poisson_pass_times(dks_poisson_plan *p, float *ms_out, int count)
{
    if (!p || !ms_out) return fail(DKS_ERR_INVALID_ARG, "plan or output pointer is NULL");
    if (p->prof_slots == 0 || p->prof_count == 0) return fail(DKS_ERR_NOT_SETUP, "no profiled solve has been issued");
    const int n = std::min(count, kNumPasses);
    const long long solves = std::min<long long>(p->prof_count, p->prof_slots);
    std::vector<double> acc(kNumPasses, 0.0);
    for (long long s = 0; s < solves; ++s) {
        cudaEvent_t *e = &p->ev[(size_t)s * prof_stride(p)];
        DKS_CUDA(cudaEventSynchronize(e[p->steps.size()]));
        for (size_t i = 0; i < p->steps.size(); ++i) {
            float ms = 0.f;
            DKS_CUDA(cudaEventElapsedTime(&ms, e[i], e[i + 1]));
            acc[p->steps[i].pass - 1] += ms;
        }
    }
    for (int i = 0; i < n; ++i) ms_out[i] = (float)(acc[i] / (double)solves);
    return n;
}

static bool last_p3(const dks_poisson_plan *p, size_t i)
{
    for (size_t j = i + 1; j < p->steps.size(); ++j) if (p->steps[j].pass == 3) return false;
    return true;
}

// Called right after the last P3 of a solve on `st`: a later rebuild of Ghat must not overtake it.
static int note_ghat_read(dks_poisson_plan *p, cudaStream_t st)
{
    if (st != p->setup_used) {
        DKS_CUDA(cudaEventRecord(p->ghat_free, st));
        p->ghat_free_recorded = true;
    } else {
        p->ghat_read_on_setup_stream = true;     // greens_setup_on records the event if the rebuild ever moves to another stream
    }
    return DKS_OK;
}

static int solve_impl(dks_poisson_plan *p, const double *rho, double *phi, int nb, void *stream)
{
    if (!p || !rho || !phi) return fail(DKS_ERR_INVALID_ARG, "plan, rho or phi is NULL");
    if (nb < 1 || nb > p->max_batch)
        return fail(DKS_ERR_INVALID_ARG, "batch of %d meshes: the plan is sized for at most %d (dks_poisson_set_max_batch)", nb, p->max_batch);
    if (p->nranks > 1) return fail(DKS_ERR_INVALID_ARG, "this plan is one rank of a sharded solve: use dks_poisson_solve_shard");
    if (nb > 1 && p->slab != p->d.nz + 1)
        return fail(DKS_ERR_INVALID_ARG, "batched solves need the default pipeline (no slabs)");
    if ((reinterpret_cast<uintptr_t>(rho) | reinterpret_cast<uintptr_t>(phi)) % 16)
        return fail(DKS_ERR_INVALID_ARG, "rho and phi must be 16-byte aligned");
    if (!p->greens_ready) return fail(DKS_ERR_NOT_SETUP, "call dks_greens_setup before dks_poisson_solve");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (p->setup_pending || st != p->setup_used) DKS_CUDA(cudaStreamIsCapturing(st, &cs));
    const bool capturing = cs != cudaStreamCaptureStatusNone;   // graph replays are ordered against dks_greens_setup by the caller
    if (p->setup_pending) {
        // Order this solve after the Green's setup.  A stream under capture must not wait on work
        // recorded outside the capture, so there the host waits for the setup instead (once).
        if (capturing) {
            cudaStreamCaptureMode mode = cudaStreamCaptureModeRelaxed;
            DKS_CUDA(cudaThreadExchangeStreamCaptureMode(&mode));
            cudaError_t e = cudaEventSynchronize(p->setup_done);
            DKS_CUDA(cudaThreadExchangeStreamCaptureMode(&mode));
            DKS_CUDA(e);
            p->setup_pending = false;
        } else {
            if (st != p->setup_used) DKS_CUDA(cudaStreamWaitEvent(st, p->setup_done, 0));
            if (cudaEventQuery(p->setup_done) == cudaSuccess) p->setup_pending = false;
            else (void)cudaGetLastError();   // cudaErrorNotReady is not a failure
        }
    }
    const bool prof = p->prof_slots > 0;
    cudaEvent_t *ev = prof ? &p->ev[(size_t)(p->prof_count % p->prof_slots) * prof_stride(p)] : nullptr;
    for (size_t i = 0; i < p->steps.size(); ++i) {
        const dks_poisson_plan::Step &s = p->steps[i];
        if (prof) DKS_CUDA(cudaEventRecord(ev[i], st));
        if (p->fast[s.pass - 1]) launch_r16(s, p, rho, phi, nb, st);
        else if (p->big[s.pass - 1] == 1024) launch_big<1024>(s, p, rho, phi, nb, st);
        else if (p->big[s.pass - 1] == 2048) launch_big<2048>(s, p, rho, phi, nb, st);
        else launch_generic(s, p, rho, phi, nb, st);
        // a later rebuild of Ghat on the setup stream must not overtake this solve's last P3
        if (s.pass == 3 && last_p3(p, i) && !capturing) {
            int rc = note_ghat_read(p, st);
            if (rc) return rc;
        }
    }
    if (prof) { DKS_CUDA(cudaEventRecord(ev[p->steps.size()], st)); ++p->prof_count; }
    DKS_CUDA(cudaGetLastError());
    return DKS_OK;
}

extern "C" int dks_poisson_solve(dks_poisson_plan *p, const double *rho, double *phi, void *stream)
{
    return solve_impl(p, rho, phi, 1, stream);
}

extern "C" int dks_poisson_solve_batch(dks_poisson_plan *p, const double *rho, double *phi, int nbatch, void *stream)
{
    return solve_impl(p, rho, phi, nbatch, stream);
}

extern "C" int dks_poisson_set_max_batch(dks_poisson_plan *p, int nbatch)
{
    if (!p) return fail(DKS_ERR_INVALID_ARG, "plan is NULL");
    if (nbatch < 1 || nbatch > 64) return fail(DKS_ERR_INVALID_ARG, "nbatch must be in [1, 64]");
    if (p->nranks > 1 && nbatch != 1) return fail(DKS_ERR_INVALID_ARG, "sharding excludes batches (this plan is rank %d of %d)", p->rank, p->nranks);
    if ((long long)(p->d.nz + 1) * nbatch > 65535)      // P2 / P4 put (plane, mesh) on gridDim.y
        return fail(DKS_ERR_INVALID_ARG, "(nz + 1) * nbatch = %lld exceeds 65535 (grid limit of the y passes)", (long long)(p->d.nz + 1) * nbatch);
    const int old = p->max_batch;
    p->max_batch = nbatch;
    compute_layout(p);
    if (p->ws && p->ws_bytes < p->need_bytes) {
        const size_t need = p->need_bytes;
        p->max_batch = old;
        compute_layout(p);
        return fail(DKS_ERR_WORKSPACE_TOO_SMALL, "the attached workspace has %zu bytes, %zu needed for batches of %d; "
                    "set the batch size before attaching the workspace / before dks_greens_setup", p->ws_bytes, need, nbatch);
    }
    p->prof_slots = 0;
    if (p->ws) { bind_workspace(p); p->greens_ready = false; }      // the Green's octant moved
    return DKS_OK;
}

extern "C" int dks_poisson_set_host_staging(dks_poisson_plan *p, int enabled)
{
    if (!p) return fail(DKS_ERR_INVALID_ARG, "plan is NULL");
    if (p->ws) return fail(DKS_ERR_INVALID_ARG, "dks_poisson_set_host_staging must be called before the workspace is attached / before dks_greens_setup");
    p->host_staging = enabled != 0;
    compute_layout(p);
    return DKS_OK;
}

// Host path.  Every call copies its rho to the device, solves and copies phi back, but consecutive calls
// overlap: the copy-in of call i+1 and the copy-out of call i-1 run on their own streams beside the solve
// of call i (PCIe is full duplex), as PAPER.md:132 does for the rho transfer.  kHostSlots staging meshes take turns.
extern "C" int dks_poisson_solve_host_async(dks_poisson_plan *p, const double *rho_host, double *phi_host, void *stream)
{
    if (!p || !rho_host || !phi_host) return fail(DKS_ERR_INVALID_ARG, "plan, rho or phi is NULL");
    if (p->nranks > 1) return fail(DKS_ERR_INVALID_ARG, "this plan is one rank of a sharded solve: it has no host path");
    if (!p->host_staging) return fail(DKS_ERR_NOT_SETUP, "the host path was switched off for this plan (dks_poisson_set_host_staging)");
    if (!p->greens_ready) return fail(DKS_ERR_NOT_SETUP, "call dks_greens_setup before dks_poisson_solve_host");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (!p->s_in) {
        DKS_CUDA(cudaStreamCreateWithFlags(&p->s_in, cudaStreamNonBlocking));
        DKS_CUDA(cudaStreamCreateWithFlags(&p->s_out, cudaStreamNonBlocking));
        for (int i = 0; i < kHostSlots; ++i) {
            DKS_CUDA(cudaEventCreateWithFlags(&p->ev_in[i], cudaEventDisableTiming));
            DKS_CUDA(cudaEventCreateWithFlags(&p->ev_solve[i], cudaEventDisableTiming));
            DKS_CUDA(cudaEventCreateWithFlags(&p->ev_out[i], cudaEventDisableTiming));
        }
    }
    const size_t bytes = sizeof(double) * (size_t)p->d.nx * p->d.ny * p->d.nz;
    const int slot = (int)(p->host_calls++ % kHostSlots);
    double *stage = p->stage + (size_t)slot * (align_up(bytes, 256) / sizeof(double));
    if (p->host_calls > (unsigned long long)kHostSlots) DKS_CUDA(cudaStreamWaitEvent(p->s_in, p->ev_out[slot], 0));   // slot free again
    DKS_CUDA(cudaMemcpyAsync(stage, rho_host, bytes, cudaMemcpyHostToDevice, p->s_in));
    DKS_CUDA(cudaEventRecord(p->ev_in[slot], p->s_in));
    DKS_CUDA(cudaStreamWaitEvent(st, p->ev_in[slot], 0));
    int rc = dks_poisson_solve(p, stage, stage, stream);
    if (rc) return rc;
    DKS_CUDA(cudaEventRecord(p->ev_solve[slot], st));
    DKS_CUDA(cudaStreamWaitEvent(p->s_out, p->ev_solve[slot], 0));
    DKS_CUDA(cudaMemcpyAsync(phi_host, stage, bytes, cudaMemcpyDeviceToHost, p->s_out));
    DKS_CUDA(cudaEventRecord(p->ev_out[slot], p->s_out));
    // later work on the caller's stream is ordered after this call's copy-out only through dks_poisson_host_sync
    return DKS_OK;
}

// One OPAL time step as PAPER.md:132 runs it: the spacings change every step, so the Green's function is
// rebuilt, on its own stream, while rho is still on its way to the device; the solve waits for both.
extern "C" int dks_poisson_step_host_async(dks_poisson_plan *p, double hx, double hy, double hz, const double *rho_host,
                                           double *phi_host, void *stream)
{
    if (!p || !rho_host || !phi_host) return fail(DKS_ERR_INVALID_ARG, "plan, rho or phi is NULL");
    int rc = dks_poisson_set_spacing(p, hx, hy, hz);
    if (rc) return rc;
    cudaStream_t ss = p->setup_stream;
    if (!ss || ss == static_cast<cudaStream_t>(stream)) {          // no stream of its own was given: use a plan-owned one
        if (!p->s_setup) DKS_CUDA(cudaStreamCreateWithFlags(&p->s_setup, cudaStreamNonBlocking));
        ss = p->s_setup;
    }
    rc = greens_setup_on(p, ss);                                    // waits for the previous step's P3, not for its P4 / P5 / copy-out
    if (rc) return rc;
    return dks_poisson_solve_host_async(p, rho_host, phi_host, stream);   // H2D on the copy stream; the solve waits for both
}

extern "C" int dks_poisson_host_sync(dks_poisson_plan *p)
{
    if (!p) return fail(DKS_ERR_INVALID_ARG, "plan is NULL");
    if (p->s_out) DKS_CUDA(cudaStreamSynchronize(p->s_out));
    return DKS_OK;
}

extern "C" int dks_poisson_solve_host(dks_poisson_plan *p, const double *rho_host, double *phi_host, void *stream)
{
    int rc = dks_poisson_solve_host_async(p, rho_host, phi_host, stream);
    if (rc) return rc;
    return dks_poisson_host_sync(p);
}

// ------------------------------------------------------------------------------------------------
// f4: the steps adjacent to the solve (dks_field_ops.cuh)
// ------------------------------------------------------------------------------------------------
static ParticleFrame frame_of(const dks_poisson_plan *p, double ox, double oy, double oz)
{
    ParticleFrame f;
    f.ox = ox; f.oy = oy; f.oz = oz; f.hx = p->hx; f.hy = p->hy; f.hz = p->hz;
    return f;
}

static int particle_grid(const dks_poisson_plan *p, long long np)
{
    const long long blocks = (np + 255) / 256;
    return (int)std::max<long long>(1, std::min<long long>(blocks, (long long)p->sm_count * 8 * 4));
}

extern "C" int dks_deposit_cic(dks_poisson_plan *p, const double *x, const double *y, const double *z, const double *q,
                               long long np, double ox, double oy, double oz, double *rho, void *stream)
{
    if (!p || !rho || np < 0 || (np > 0 && (!x || !y || !z || !q))) return fail(DKS_ERR_INVALID_ARG, "plan, rho or a particle array is NULL, or np < 0");
    if (!std::isfinite(ox) || !std::isfinite(oy) || !std::isfinite(oz)) return fail(DKS_ERR_INVALID_ARG, "origin must be finite");
    int rc = ensure_device(p);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t nodes = (size_t)p->d.nx * p->d.ny * p->d.nz;
    DKS_CUDA(cudaMemsetAsync(rho, 0, sizeof(double) * nodes, st));
    if (np > 0)
        cic_deposit_kernel<<<particle_grid(p, np), 256, 0, st>>>(x, y, z, q, np, frame_of(p, ox, oy, oz), p->d,
                                                                  1.0 / (p->hx * p->hy * p->hz), rho);
    DKS_CUDA(cudaGetLastError());
    return DKS_OK;
}

extern "C" int dks_gradient(dks_poisson_plan *p, const double *phi, double *ex, double *ey, double *ez, void *stream)
{
    if (!p || !phi || !ex || !ey || !ez) return fail(DKS_ERR_INVALID_ARG, "plan or a field pointer is NULL");
    if (phi == ex || phi == ey || phi == ez) return fail(DKS_ERR_INVALID_ARG, "the field components must not alias phi");
    int rc = ensure_device(p);
    if (rc) return rc;
    const MeshDims d = p->d;
    gradient_kernel<<<dim3((d.nx + 127) / 128, d.ny, d.nz), 128, 0, static_cast<cudaStream_t>(stream)>>>(
        phi, ex, ey, ez, d, 0.5 / p->hx, 0.5 / p->hy, 0.5 / p->hz);
    DKS_CUDA(cudaGetLastError());
    return DKS_OK;
}

extern "C" int dks_gather_field(dks_poisson_plan *p, const double *ex, const double *ey, const double *ez, const double *x,
                                const double *y, const double *z, long long np, double ox, double oy, double oz,
                                double *epx, double *epy, double *epz, void *stream)
{
    if (!p || !ex || !ey || !ez || np < 0 || (np > 0 && (!x || !y || !z || !epx || !epy || !epz)))
        return fail(DKS_ERR_INVALID_ARG, "plan, a field or a particle array is NULL, or np < 0");
    if (!std::isfinite(ox) || !std::isfinite(oy) || !std::isfinite(oz)) return fail(DKS_ERR_INVALID_ARG, "origin must be finite");
    int rc = ensure_device(p);
    if (rc) return rc;
    if (np > 0)
        gather_field_kernel<<<particle_grid(p, np), 256, 0, static_cast<cudaStream_t>(stream)>>>(ex, ey, ez, x, y, z, np,
                                                                                                  frame_of(p, ox, oy, oz), p->d, epx, epy, epz);
    DKS_CUDA(cudaGetLastError());
    return DKS_OK;
}

// dks_gradient followed by dks_gather_field without the three field meshes: the field lives for the duration of the call in the
// plan's buffer B (free between solves), interleaved (dks_field_ops.cuh).
extern "C" int dks_field_at_particles(dks_poisson_plan *p, const double *phi, const double *x, const double *y, const double *z,
                                      long long np, double ox, double oy, double oz, double *epx, double *epy, double *epz, void *stream)
{
    if (!p || !phi || np < 0 || (np > 0 && (!x || !y || !z || !epx || !epy || !epz)))
        return fail(DKS_ERR_INVALID_ARG, "plan, phi or a particle array is NULL, or np < 0");
    if (!std::isfinite(ox) || !std::isfinite(oy) || !std::isfinite(oz)) return fail(DKS_ERR_INVALID_ARG, "origin must be finite");
    if (!p->ws || !p->B) return fail(DKS_ERR_NOT_SETUP, "dks_field_at_particles uses the plan's workspace: attach one or call dks_greens_setup first");
    if (p->nranks > 1 || p->slab != p->d.nz + 1)
        return fail(DKS_ERR_INVALID_ARG, "dks_field_at_particles needs the full buffer B: not available on slabbed or sharded plans");
    int rc = ensure_device(p);
    if (rc) return rc;
    if (np == 0) return DKS_OK;
    const MeshDims d = p->d;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    double4 *e = reinterpret_cast<double4 *>(p->B);            // 32 nx ny nz bytes <= 32 nx ny (nz + 1) = sizeof B
    gradient_aos_kernel<<<dim3((d.nx + 127) / 128, d.ny, d.nz), 128, 0, st>>>(phi, e, d, 0.5 / p->hx, 0.5 / p->hy, 0.5 / p->hz);
    gather_aos_kernel<<<particle_grid(p, np), 256, 0, st>>>(e, x, y, z, np, frame_of(p, ox, oy, oz), d, epx, epy, epz);
    DKS_CUDA(cudaGetLastError());
    return DKS_OK;
}

// ------------------------------------------------------------------------------------------------
// f3: one solve sharded over several GPUs; DESIGN.md section 9
// ------------------------------------------------------------------------------------------------
extern "C" int dks_poisson_set_shard(dks_poisson_plan *p, int rank, int nranks)
{
    if (!p) return fail(DKS_ERR_INVALID_ARG, "plan is NULL");
    if (nranks < 1 || nranks > kMaxRanks || (nranks & (nranks - 1)) || rank < 0 || rank >= nranks)
        return fail(DKS_ERR_INVALID_ARG, "nranks must be a power of two in [1, %d] and 0 <= rank < nranks", kMaxRanks);
    if (p->ws) return fail(DKS_ERR_INVALID_ARG, "dks_poisson_set_shard must be called before the workspace is attached / before dks_greens_setup");
    if (nranks > 1) {
        if (!(p->fast[0] && p->fast[1] && p->fast[2]))
            return fail(DKS_ERR_INVALID_ARG, "a sharded solve needs nx, ny, nz in [16, 256] (register-resident passes on every axis)");
        if (p->d.ny / nranks < 1 || p->d.nz / nranks < 1) return fail(DKS_ERR_INVALID_ARG, "more ranks than rows");
        if (p->max_batch != 1 || p->slab != p->d.nz + 1) return fail(DKS_ERR_INVALID_ARG, "sharding excludes batches and slabs");
    }
    p->rank = rank; p->nranks = nranks;
    p->ny_loc = p->d.ny / nranks; p->y0 = rank * p->ny_loc;
    const int split = p->d.nz / nranks;                       // the last rank also takes plane nz
    p->kz0 = rank * split; p->planes_loc = split + (rank == nranks - 1 ? 1 : 0);
    p->pdl = p->pdl && nranks == 1;
    compute_layout(p);
    return DKS_OK;
}

extern "C" int dks_poisson_shard_buffers(dks_poisson_plan *p, void **recv_p1, void **recv_p4)
{
    if (!p || !recv_p1 || !recv_p4) return fail(DKS_ERR_INVALID_ARG, "plan or output pointer is NULL");
    if (p->nranks < 2 || !p->ws) return fail(DKS_ERR_NOT_SETUP, "call dks_poisson_set_shard and attach the workspace (or dks_greens_setup) first");
    *recv_p1 = p->A; *recv_p4 = p->A2;
    return DKS_OK;
}

extern "C" int dks_poisson_set_peers(dks_poisson_plan *p, void *const *recv_p1_of_rank, void *const *recv_p4_of_rank)
{
    if (!p || !recv_p1_of_rank || !recv_p4_of_rank) return fail(DKS_ERR_INVALID_ARG, "plan or pointer table is NULL");
    if (p->nranks < 2 || !p->ws) return fail(DKS_ERR_NOT_SETUP, "call dks_poisson_set_shard and attach the workspace (or dks_greens_setup) first");
    int l1 = 0, l2 = 0;
    while ((1 << l1) < p->d.nz / p->nranks) ++l1;
    while ((1 << l2) < p->ny_loc) ++l2;
    for (int r = 0; r < p->nranks; ++r) {
        if (!recv_p1_of_rank[r] || !recv_p4_of_rank[r]) return fail(DKS_ERR_INVALID_ARG, "peer buffer of rank %d is NULL", r);
        p->peers1.base[r] = static_cast<cplx *>(recv_p1_of_rank[r]);
        p->peers2.base[r] = static_cast<cplx *>(recv_p4_of_rank[r]);
    }
    if (p->peers1.base[p->rank] != p->A || p->peers2.base[p->rank] != p->A2)
        return fail(DKS_ERR_INVALID_ARG, "entry %d of the tables must be this rank's own buffers (dks_poisson_shard_buffers)", p->rank);
    p->peers1.nranks = p->peers2.nranks = p->nranks;
    p->peers1.lsplit = l1; p->peers1.first = p->y0; p->peers1.pitch = p->d.ny;
    p->peers2.lsplit = l2; p->peers2.first = p->kz0; p->peers2.pitch = p->ny_loc;
    p->peers_set = true;
    return DKS_OK;
}

template <int A>
static void shard_launch_p1(const dks_poisson_plan *p, const double *rho, cudaStream_t st)
{
    MeshDims d = p->d;
    d.ny = p->ny_loc;                                          // this rank's y rows only
    const int T = R16Geom<A>::THREADS, tiles = d.nx / (2 * kCols) * d.ny;
    const int per_sm = std::max(1, std::min(512 / T, (227 * 1024) / (P1Geom<A>::SMEM + 1024)));
    p1_z_r2c_r16<A, false, true><<<std::min(tiles, p->sm_count * per_sm), T, P1Geom<A>::SMEM, st>>>(rho, nullptr, d, 1, p->tw1[2], p->tw[2], p->peers1);
}

template <int A>
static void shard_launch_p4(const dks_poisson_plan *p, cudaStream_t st)
{
    p4_y_inv_r16<A, false, true><<<dim3(p->d.nx / kCols, p->planes_loc), R16Geom<A>::THREADS, R16Geom<A>::SMEM, st>>>(
        p->B, nullptr, p->d, 0, p->tw1[1], p->tw[1], p->peers2);
}

// phase 1: P1 on this rank's y slab, rows stored to the owners of their kz planes
// phase 2: P2, P3, P4 on this rank's kz slab, P4's rows stored to the owners of their y rows
// phase 3: P5 on this rank's y slab
// Between the phases every rank must have finished the previous phase (the caller's barrier: an NCCL barrier on the same
// stream, or stream order when the ranks are emulated on one device).
extern "C" int dks_poisson_solve_shard(dks_poisson_plan *p, int phase, const double *rho_loc, double *phi_loc, void *stream)
{
    if (!p) return fail(DKS_ERR_INVALID_ARG, "plan is NULL");
    if (p->nranks < 2 || !p->peers_set) return fail(DKS_ERR_NOT_SETUP, "call dks_poisson_set_shard, dks_greens_setup and dks_poisson_set_peers first");
    if (!p->greens_ready) return fail(DKS_ERR_NOT_SETUP, "call dks_greens_setup before dks_poisson_solve_shard");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (p->setup_pending && st != p->setup_used) DKS_CUDA(cudaStreamWaitEvent(st, p->setup_done, 0));
    const MeshDims d = p->d;
    switch (phase) {
    case 1:
        if (!rho_loc || reinterpret_cast<uintptr_t>(rho_loc) % 16) return fail(DKS_ERR_INVALID_ARG, "rho_loc is NULL or not 16-byte aligned");
        switch (p->r16A[2]) {
#define X(A_) case A_: shard_launch_p1<A_>(p, rho_loc, st); break;
            DKS_FOR_EACH_A(X)
#undef X
        }
        break;
    case 2: {
        dks_poisson_plan::Step s2 = { 2, 0, p->planes_loc }, s3 = { 3, p->kz0, p->planes_loc };
        launch_r16(s2, p, nullptr, nullptr, 1, st);            // reads A1 (= p->A, local planes), writes B
        launch_r16(s3, p, nullptr, nullptr, 1, st);            // Ghat planes kz0 ..
        { int rc = note_ghat_read(p, st); if (rc) return rc; }
        switch (p->r16A[1]) {
#define X(A_) case A_: shard_launch_p4<A_>(p, st); break;
            DKS_FOR_EACH_A(X)
#undef X
        }
        break;
    }
    case 3: {
        if (!phi_loc || reinterpret_cast<uintptr_t>(phi_loc) % 16) return fail(DKS_ERR_INVALID_ARG, "phi_loc is NULL or not 16-byte aligned");
        MeshDims dl = d;
        dl.ny = p->ny_loc;
        switch (p->r16A[2]) {
#define X(A_) case A_: p5_z_c2r_r16<A_, false><<<dim3(d.nx / (2 * kCols), dl.ny, 1), R16Geom<A_>::THREADS, R16Geom<A_>::SMEM, st>>>(p->A2, phi_loc, dl, p->tw1[2], p->tw[2]); break;
            DKS_FOR_EACH_A(X)
#undef X
        }
        break;
    }
    default: return fail(DKS_ERR_INVALID_ARG, "phase must be 1, 2 or 3");
    }
    DKS_CUDA(cudaGetLastError());
    return DKS_OK;
}

// ------------------------------------------------------------------------------------------------
// dks_field_at_particles_static: the field at the particles for callers that cannot allocate device memory
// ------------------------------------------------------------------------------------------------
// dks_field_at_particles keeps the node field (one 32-byte record per node) in the plan's buffer B, and a plan means
// cudaMalloc: the twiddle tables on first use, and the workspace unless the caller brings one.  Some users of this
// library cannot go there.  Examples: a tracking loop in which a cudaMalloc or cudaFree would stall every other stream
// of the process (both synchronise the whole device); a host code whose own pool has already reserved all device
// memory, so that a fresh cudaMalloc simply fails; a plug-in that is handed device pointers by its host and owns no
// allocator.  For them the record array below lives in the library image itself.  Its price: every GPU on which this
// library's module gets loaded holds these 8 MiB until the process exits, used or not, which is why the limit is modest.
//
// g_field_scratch is a __device__ symbol.  In host code its name is a host-side shadow, NOT a device address (a kernel
// handed &g_field_scratch from the host would fault, or on systems where the GPU can reach host memory scribble over
// host memory), so the host asks the runtime for the address, once per device and with that device current.
static __device__ __align__(256) double g_field_scratch[4 * (size_t)DKS_STATIC_FIELD_MAX_NODES];

static const int kStaticMaxDevices = 64;
struct StaticScratchSlot { double4 *ptr = nullptr; int sm_count = 0; bool ready = false; };
static StaticScratchSlot g_static_slot[kStaticMaxDevices];
static std::mutex g_static_mutex;

// Set-up of the current device, done by the first call on it: architecture check, SM count, device address of the array.
// Neither call below allocates (the array came with the module).
static int static_scratch_of_current_device(StaticScratchSlot *out)
{
    int dev = -1;
    DKS_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return fail(DKS_ERR_UNSUPPORTED_DEVICE, "device ordinal %d is outside [0, %d)", dev, kStaticMaxDevices);
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticScratchSlot &s = g_static_slot[dev];
    if (!s.ready) {
        int major = 0, sms = 0;
        DKS_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        DKS_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        if (major != 10)
            return fail(DKS_ERR_UNSUPPORTED_DEVICE, "device %d is compute capability %d.x; this library is built for sm_100a only", dev, major);
        void *addr = nullptr;
        DKS_CUDA(cudaGetSymbolAddress(&addr, g_field_scratch));
        if (!addr || reinterpret_cast<uintptr_t>(addr) % 256) return fail(DKS_ERR_CUDA, "cudaGetSymbolAddress gave %p for the field scratch", addr);
        s.ptr = static_cast<double4 *>(addr); s.sm_count = sms; s.ready = true;
    }
    *out = s;
    return DKS_OK;
}

extern "C" int dks_field_at_particles_static(int nx, int ny, int nz, double hx, double hy, double hz, const double *phi,
                                             const double *x, const double *y, const double *z, long long np, double ox, double oy,
                                             double oz, double *epx, double *epy, double *epz, void *stream)
{
    if (!is_pow2_in_range(nx) || !is_pow2_in_range(ny) || !is_pow2_in_range(nz))
        return fail(DKS_ERR_INVALID_ARG, "mesh %dx%dx%d: every extent must be a power of two in [8, 1024]", nx, ny, nz);
    const long long nodes = (long long)nx * ny * nz;
    if (nodes > (long long)DKS_STATIC_FIELD_MAX_NODES)
        return fail(DKS_ERR_INVALID_ARG, "mesh %dx%dx%d has %lld nodes; dks_field_at_particles_static holds at most %lld "
                    "(DKS_STATIC_FIELD_MAX_NODES, e.g. 64x64x64): use dks_field_at_particles with a plan for larger meshes",
                    nx, ny, nz, nodes, (long long)DKS_STATIC_FIELD_MAX_NODES);
    if (!(hx > 0) || !(hy > 0) || !(hz > 0) || !std::isfinite(hx) || !std::isfinite(hy) || !std::isfinite(hz))
        return fail(DKS_ERR_INVALID_ARG, "spacings must be finite and > 0 (got %g, %g, %g)", hx, hy, hz);
    if (!phi || np < 0 || (np > 0 && (!x || !y || !z || !epx || !epy || !epz)))
        return fail(DKS_ERR_INVALID_ARG, "phi or a particle array is NULL, or np < 0");
    if (!std::isfinite(ox) || !std::isfinite(oy) || !std::isfinite(oz)) return fail(DKS_ERR_INVALID_ARG, "origin must be finite");
    StaticScratchSlot s;
    int rc = static_scratch_of_current_device(&s);
    if (rc) return rc;
    if (np == 0) return DKS_OK;
    MeshDims d = MeshDims();                                   // the two kernels read nx, ny, nz only
    d.nx = nx; d.ny = ny; d.nz = nz;
    ParticleFrame f;
    f.ox = ox; f.oy = oy; f.oz = oz; f.hx = hx; f.hy = hy; f.hz = hz;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // Nothing in the array has to start at zero: the first kernel writes the record of every node of this mesh and the
    // second reads only those, so whatever the previous call (of any mesh shape) left behind is never seen.
    gradient_aos_kernel<<<dim3((nx + 127) / 128, ny, nz), 128, 0, st>>>(phi, s.ptr, d, 0.5 / hx, 0.5 / hy, 0.5 / hz);
    const long long blocks = (np + 255) / 256;
    const int grid = (int)std::max<long long>(1, std::min<long long>(blocks, (long long)s.sm_count * 8 * 4));
    gather_aos_kernel<<<grid, 256, 0, st>>>(s.ptr, x, y, z, np, f, d, epx, epy, epz);
    DKS_CUDA(cudaGetLastError());
    return DKS_OK;
}

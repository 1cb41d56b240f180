// grx_api.cu -- the C ABI of include/grx.h: argument validation on the host, launch geometry, error mapping.
// No torch types, no allocation of user memory; state: the kernel selector, the per-thread debug counter pointer and
// the per-thread streams of the host entry point (include/grx.h, "State").
#include <atomic>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

#include "../../include/grx.h"
#include "grx_launch.h"

namespace {

thread_local char t_err[256] = "";
thread_local unsigned long long* t_fallback_counter = nullptr;
std::atomic<int> g_variant{GRX_VARIANT_AUTO};

int fail(int code, const char* msg) {
    std::snprintf(t_err, sizeof(t_err), "%s", msg);
    return code;
}
int fail_cuda(cudaError_t e, const char* where) {
    std::snprintf(t_err, sizeof(t_err), "%s: %s", where, cudaGetErrorString(e));
    return GRX_ERR_CUDA;
}

// Fills the geometry part of RhsParams; returns nullptr if fine, else what is wrong.
const char* make_geom(const grx_grid* grid, int nghost, grx::RhsParams& p) {
    if (!grid) return "grid is NULL";
    if (grid->nx < 1 || grid->ny < 1 || grid->nz < 1) return "grid: nx, ny, nz must be >= 1";
    if (grid->nbox < 1 || grid->nbox > 65535) return "grid: nbox must be in [1, 65535]";
    if (nghost < 0 || nghost > 1024) return "nghost out of range";
    p.n[0] = grid->nx; p.n[1] = grid->ny; p.n[2] = grid->nz;
    long long nc = 1;
    for (int a = 0; a < 3; ++a) {
        p.N[a] = p.n[a] + 2 * nghost;
        nc *= p.N[a];
        if (nc > 2147483647LL) return "a box (with ghosts) must not exceed 2^31-1 cells";
    }
    p.g = nghost;
    p.nbox = grid->nbox;
    p.nc = nc;
    p.stride[0] = 1;
    p.stride[1] = p.N[0];
    p.stride[2] = (long long)p.N[0] * p.N[1];
    return nullptr;
}

// Kernel of the product path for this block: 0 = simple, 1 = LDG, 2 = TMA, -1 = TMA forced on arrays it cannot take.
int choose_kernel(const grx::RhsParams& p, int recon) {
    const int variant = g_variant.load();
    if (variant == GRX_VARIANT_SIMPLE) return 0;
    if (variant == GRX_VARIANT_LDG) return 1;
    const bool ok = grx::tma_supported(p);
    if (variant == GRX_VARIANT_TMA) return ok ? 2 : -1;
    if (!ok) return 1;
    // AUTO, both kernels take the block: choose by the expected time.  Per cell of a well-filled machine the TMA kernel
    // is about 1.12x (WENO5) to 1.22x (TVD) faster; on small blocks and batches its 7-row tiles and its per-chunk
    // set-up fill the SMs less well than the LDG kernel's 11-row tiles (constants fitted on the config-5 sweep,
    // profiles/r2_sweep.md: the selector picks the faster kernel at every point).
    int dev = 0, sms = 0;
    if (grx::current_device_sms(&dev, &sms) == cudaSuccess) {
        const double gain = (recon == GRX_RECON_WENO5) ? 1.12 : 1.22;
        if (gain * grx::tma_tile_efficiency(p, sms) < grx::fused_tile_efficiency(p, sms)) return 1;
    }
    return 2;
}

// Launches the selected kernel on a (sub-)block.  `unsupported` is set when the TMA kernel was forced on arrays it
// cannot take.
cudaError_t launch_variant(const grx::RhsParams& p, int recon, cudaStream_t st, bool* unsupported = nullptr) {
    switch (choose_kernel(p, recon)) {
        case 0: return grx::launch_rhs_simple(p, recon, st);
        case 1: return grx::launch_rhs_fused(p, recon, st);
        case 2: return grx::launch_rhs_tma(p, recon, 7, st);
        default:
            if (unsupported) *unsupported = true;
            return cudaErrorNotSupported;
    }
}

// Launches kernel `kernel` (a choose_kernel result >= 0 taken on the WHOLE block) on a block or on a z sub-block of it.
// nz_whole: interior planes of the whole block -- the LDG kernel picks its row tile from it, so that every plane of a
// sub-block carries the bits of the whole-block call (the two kernels, and the tiles of one, round differently).
cudaError_t launch_chosen(int kernel, const grx::RhsParams& p, int recon, cudaStream_t st, int nz_whole) {
    return kernel == 0 ? grx::launch_rhs_simple(p, recon, st)
         : kernel == 1 ? grx::launch_rhs_fused(p, recon, st, nz_whole) : grx::launch_rhs_tma(p, recon, 7, st);
}

// The two internal streams of grx_valencia_rhs_host: one pair per host thread and device, created on first use.
struct HostStreams {
    int dev = -1;
    cudaStream_t up = nullptr, dn = nullptr;
    ~HostStreams() {
        // At thread exit the context may already be gone: errors are ignored.
        if (up) cudaStreamDestroy(up);
        if (dn) cudaStreamDestroy(dn);
    }
};
cudaError_t host_streams(cudaStream_t* up, cudaStream_t* dn) {
    thread_local std::vector<HostStreams> pool;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    for (HostStreams& h : pool)
        if (h.dev == dev) { *up = h.up; *dn = h.dn; return cudaSuccess; }
    pool.emplace_back();
    HostStreams& h = pool.back();
    h.dev = dev;
    e = cudaStreamCreateWithFlags(&h.up, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&h.dn, cudaStreamNonBlocking);
    if (e != cudaSuccess) { pool.pop_back(); return e; }
    *up = h.up; *dn = h.dn;
    return cudaSuccess;
}

// Right-hand side with constrained transport (NEXT-2): p.fb is set.  The TMA kernel writes the face fluxes of the interior
// grid lines while it evaluates the right-hand side; the other kernels do not, and then every face is evaluated by the
// face kernel.  Same kernel choice as grx_valencia_rhs, so that out[0..4] are its bits.
cudaError_t launch_rhs_ct(grx::RhsParams p, int recon, cudaStream_t st, bool* unsupported) {
    const int kernel = choose_kernel(p, recon);
    if (kernel < 0) {
        if (unsupported) *unsupported = true;
        return cudaErrorNotSupported;
    }
    const bool fused_faces = (kernel == 2);
    cudaError_t e;
    if (fused_faces) {
        e = grx::launch_rhs_tma(p, recon, 7, st);
    } else {
        grx::RhsParams q = p;
        q.fb = nullptr;
        e = launch_variant(q, recon, st);
    }
    p.nfallback = nullptr;   // the faces next to the block are not faces of the right-hand side: not counted
    if (e == cudaSuccess) e = grx::launch_face_bflux(p, recon, !fused_faces, st);
    if (e == cudaSuccess) e = grx::launch_flux_ct(p, st);
    return e;
}

// ---- grx_valencia_rhs_ct_static: the face-flux scratch of constrained transport as part of the library image ----------
// For callers that cannot allocate device memory (include/grx.h says who and why).  The array below lives in the device
// image of this translation unit: every device that loads the library carries its 16 MiB until the process ends.
// In host code the NAME of a __device__ array is only a handle for the runtime -- it is not an address the GPU can use; a
// kernel handed `g_ct_static_scratch` from the host would fault or scribble over unrelated memory.  The device address
// comes from cudaGetSymbolAddress, asked once per device with that device current, and is what the kernels receive.
constexpr size_t CT_STATIC_DOUBLES = GRX_CT_STATIC_MAX_BYTES / sizeof(double);
static __device__ __align__(256) double g_ct_static_scratch[CT_STATIC_DOUBLES];

constexpr int CT_STATIC_MAX_DEVICES = 64;
std::mutex g_ct_static_mutex;
double* g_ct_static_addr[CT_STATIC_MAX_DEVICES] = {};   // device address of the array on device i, nullptr = not asked yet

// Device address of the scratch array on the calling thread's current device (looked up on the first call per device).
cudaError_t ct_static_scratch(double** addr) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= CT_STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_ct_static_mutex);
    if (!g_ct_static_addr[dev]) {
        void* a = nullptr;
        e = cudaGetSymbolAddress(&a, g_ct_static_scratch);
        if (e != cudaSuccess) return e;
        if (!a) return cudaErrorInvalidSymbol;
        g_ct_static_addr[dev] = static_cast<double*>(a);
    }
    *addr = g_ct_static_addr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" {

int grx_valencia_rhs(const grx_grid* grid, const double* prim, const double* metric, const double* K,
                     const double dx[3], int nghost, int recon, double gamma, double* out, void* cuda_stream) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (const char* why = make_geom(grid, nghost, p)) return fail(GRX_ERR_INVALID_ARG, why);
    if (!prim || !metric || !K || !dx || !out) return fail(GRX_ERR_INVALID_ARG, "NULL array pointer");
    if (recon != GRX_RECON_MINMOD && recon != GRX_RECON_MC && recon != GRX_RECON_WENO5)
        return fail(GRX_ERR_INVALID_ARG, "unknown recon");
    if (nghost < (recon == GRX_RECON_WENO5 ? 3 : 2))
        return fail(GRX_ERR_INVALID_ARG, "nghost too small: WENO5 needs 3, minmod/MC need 2 (R29)");
    if (!(gamma > 1.0)) return fail(GRX_ERR_INVALID_ARG, "gamma must be > 1");
    for (int a = 0; a < 3; ++a) {
        if (!(dx[a] > 0.0) || !(1.0 / dx[a] > 0.0)) return fail(GRX_ERR_INVALID_ARG, "dx must be > 0 and finite");
        p.idx[a] = 1.0 / dx[a];
    }
    if (out == prim || out == metric || out == K) return fail(GRX_ERR_INVALID_ARG, "out must not alias an input");
    p.prim = prim; p.met = metric; p.K = K; p.out = out;
    p.gamma = gamma;
    p.nfallback = t_fallback_counter;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    bool unsupported = false;
    const cudaError_t e = launch_variant(p, recon, st, &unsupported);
    if (unsupported) return fail(GRX_ERR_UNSUPPORTED, "GRX_VARIANT_TMA needs even nx + 2 nghost and 16-byte aligned arrays");
    if (e != cudaSuccess) return fail_cuda(e, "grx_valencia_rhs launch");
    return GRX_OK;
}

size_t grx_host_workspace_bytes(const grx_grid* grid, int nghost) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (make_geom(grid, nghost, p)) return 0;
    return (size_t)32 * (size_t)p.nc * (size_t)p.nbox * sizeof(double);
}

int grx_valencia_rhs_host(const grx_grid* grid, const double* prim_host, const double* metric_host,
                          const double* K_host, const double dx[3], int nghost, int recon, double gamma,
                          double* out_host, void* workspace, size_t workspace_bytes, void* cuda_stream) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (const char* why = make_geom(grid, nghost, p)) return fail(GRX_ERR_INVALID_ARG, why);
    if (!prim_host || !metric_host || !K_host || !out_host || !workspace || !dx)
        return fail(GRX_ERR_INVALID_ARG, "NULL array pointer");
    if (recon != GRX_RECON_MINMOD && recon != GRX_RECON_MC && recon != GRX_RECON_WENO5)
        return fail(GRX_ERR_INVALID_ARG, "unknown recon");
    if (nghost < (recon == GRX_RECON_WENO5 ? 3 : 2))
        return fail(GRX_ERR_INVALID_ARG, "nghost too small: WENO5 needs 3, minmod/MC need 2 (R29)");
    if (!(gamma > 1.0)) return fail(GRX_ERR_INVALID_ARG, "gamma must be > 1");
    for (int a = 0; a < 3; ++a) {
        if (!(dx[a] > 0.0) || !(1.0 / dx[a] > 0.0)) return fail(GRX_ERR_INVALID_ARG, "dx must be > 0 and finite");
        p.idx[a] = 1.0 / dx[a];
    }
    const size_t cells = (size_t)p.nc * (size_t)p.nbox;
    if (workspace_bytes < 32 * cells * sizeof(double)) return fail(GRX_ERR_INVALID_ARG, "workspace too small");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    double* d_prim = static_cast<double*>(workspace);
    double* d_met = d_prim + 8 * cells;
    double* d_K = d_met + 10 * cells;
    double* d_out = d_K + 6 * cells;
    p.prim = d_prim; p.met = d_met; p.K = d_K; p.out = d_out;
    p.gamma = gamma;
    p.nfallback = t_fallback_counter;

    // Slab pipeline along z: the upload of planes [j*CH, (j+1)*CH) runs on its own stream; slab i (interior
    // planes [i*CH, (i+1)*CH)) is evaluated on the caller's stream as soon as the planes it reads (up to
    // (i+1)*CH + 2g - 1) have arrived; its result goes back on a third stream.  H2D, kernels and D2H overlap;
    // every cell sees the same arithmetic as in the single-launch path (bitwise identical results).
    const int CH = 32;
    const int Nz = p.N[2], nz = p.n[2], g = p.g;
    const bool pipelined = (nz > CH) && (2 * g <= CH) && (t_fallback_counter == nullptr);
    if (!pipelined) {
        cudaError_t e = cudaMemcpyAsync(d_prim, prim_host, 8 * cells * sizeof(double), cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(d_met, metric_host, 10 * cells * sizeof(double), cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(d_K, K_host, 6 * cells * sizeof(double), cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return fail_cuda(e, "grx_valencia_rhs_host H2D");
        e = launch_variant(p, recon, st);
        if (e != cudaSuccess) return fail_cuda(e, "grx_valencia_rhs_host launch");
        e = cudaMemcpyAsync(out_host, d_out, 8 * cells * sizeof(double), cudaMemcpyDeviceToHost, st);
        if (e != cudaSuccess) return fail_cuda(e, "grx_valencia_rhs_host D2H");
        return GRX_OK;
    }
    // One kernel choice for all slabs, taken on the whole block as the device entry point takes it: the selector looks at
    // the geometry (a 32-plane slab fills the machine differently from the block), and results must not depend on it.
    const int kernel = choose_kernel(p, recon);
    if (kernel < 0) return fail(GRX_ERR_UNSUPPORTED, "GRX_VARIANT_TMA needs even nx + 2 nghost and 16-byte aligned arrays");
    cudaStream_t s_up = nullptr, s_dn = nullptr;
    cudaEvent_t ev_start = nullptr, ev_dn = nullptr;
    // a tail shorter than 8 planes joins the last full slab (no slab thinner than the stencil work it amortises)
    const int nchunk = (Nz + CH - 1) / CH, nslab = (nz % CH != 0 && nz % CH < 8) ? nz / CH : (nz + CH - 1) / CH;
    std::vector<cudaEvent_t> ev_up(nchunk, nullptr), ev_done(nslab, nullptr);
    cudaError_t e = host_streams(&s_up, &s_dn);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ev_start, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ev_dn, cudaEventDisableTiming);
    for (int j = 0; j < nchunk && e == cudaSuccess; ++j) e = cudaEventCreateWithFlags(&ev_up[j], cudaEventDisableTiming);
    for (int i = 0; i < nslab && e == cudaSuccess; ++i) e = cudaEventCreateWithFlags(&ev_done[i], cudaEventDisableTiming);
    const size_t plane = (size_t)p.stride[2];
    // the workspace may still be in use by earlier work on the caller's stream
    if (e == cudaSuccess) e = cudaEventRecord(ev_start, st);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(s_up, ev_start, 0);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(s_dn, ev_start, 0);
    struct Arr { const double* h; double* d; int nf; };
    const Arr in[3] = {{prim_host, d_prim, 8}, {metric_host, d_met, 10}, {K_host, d_K, 6}};
    int uploaded = 0;   // chunks enqueued so far
    auto upload_to = [&](int last_chunk) {
        for (; uploaded <= last_chunk && uploaded < nchunk && e == cudaSuccess; ++uploaded) {
            const int z0 = uploaded * CH, z1 = (z0 + CH < Nz) ? z0 + CH : Nz;
            const size_t off = (size_t)z0 * plane, bytes = (size_t)(z1 - z0) * plane * sizeof(double);
            for (int a = 0; a < 3 && e == cudaSuccess; ++a)
                for (int bf = 0; bf < p.nbox * in[a].nf && e == cudaSuccess; ++bf)
                    e = cudaMemcpyAsync(in[a].d + (size_t)bf * p.nc + off, in[a].h + (size_t)bf * p.nc + off, bytes,
                                        cudaMemcpyHostToDevice, s_up);
            if (e == cudaSuccess) e = cudaEventRecord(ev_up[uploaded], s_up);
        }
    };
    for (int i = 0; i < nslab && e == cudaSuccess; ++i) {
        const int k0 = i * CH, k1 = (i == nslab - 1) ? nz : k0 + CH;
        const int need = (k1 + 2 * g - 1) / CH;                   // last chunk this slab reads
        upload_to(need + 1);                                      // keep one chunk of upload ahead of the kernels
        if (e != cudaSuccess) break;
        e = cudaStreamWaitEvent(st, ev_up[need < nchunk ? need : nchunk - 1], 0);
        if (e != cudaSuccess) break;
        grx::RhsParams ps = p;
        const size_t off = (size_t)k0 * plane;
        ps.prim = d_prim + off; ps.met = d_met + off; ps.K = d_K + off; ps.out = d_out + off;
        ps.n[2] = k1 - k0;
        ps.N[2] = (k1 - k0) + 2 * g;
        e = launch_chosen(kernel, ps, recon, st, nz);
        if (e == cudaSuccess) e = cudaEventRecord(ev_done[i], st);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(s_dn, ev_done[i], 0);
        const size_t ooff = (size_t)(k0 + g) * plane, obytes = (size_t)(k1 - k0) * plane * sizeof(double);
        for (int bf = 0; bf < p.nbox * 8 && e == cudaSuccess; ++bf)
            e = cudaMemcpyAsync(out_host + (size_t)bf * p.nc + ooff, d_out + (size_t)bf * p.nc + ooff, obytes,
                                cudaMemcpyDeviceToHost, s_dn);
    }
    upload_to(nchunk - 1);
    // the caller's stream is done when the last download is
    if (e == cudaSuccess) e = cudaEventRecord(ev_dn, s_dn);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(st, ev_dn, 0);
    if (e == cudaSuccess) e = cudaEventRecord(ev_dn, s_up);      // and the (already drained) upload stream
    if (e == cudaSuccess) e = cudaStreamWaitEvent(st, ev_dn, 0);
    for (cudaEvent_t ev : ev_up) if (ev) cudaEventDestroy(ev);
    for (cudaEvent_t ev : ev_done) if (ev) cudaEventDestroy(ev);
    if (ev_start) cudaEventDestroy(ev_start);
    if (ev_dn) cudaEventDestroy(ev_dn);
    if (e != cudaSuccess) return fail_cuda(e, "grx_valencia_rhs_host pipeline");
    return GRX_OK;
}

int grx_prim2con(const grx_grid* grid, const double* prim, const double* metric, int nghost, double gamma,
                 double* cons, void* cuda_stream) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (const char* why = make_geom(grid, nghost, p)) return fail(GRX_ERR_INVALID_ARG, why);
    if (!prim || !metric || !cons) return fail(GRX_ERR_INVALID_ARG, "NULL array pointer");
    if (!(gamma > 1.0)) return fail(GRX_ERR_INVALID_ARG, "gamma must be > 1");
    const cudaError_t e = grx::launch_prim2con(prim, metric, p.nc, p.nbox, gamma, cons, static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return fail_cuda(e, "grx_prim2con launch");
    return GRX_OK;
}

int grx_con2prim(const grx_grid* grid, const double* cons, const double* metric, int nghost, double gamma,
                 double* prim, unsigned long long* nfail, void* cuda_stream) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (const char* why = make_geom(grid, nghost, p)) return fail(GRX_ERR_INVALID_ARG, why);
    if (!prim || !metric || !cons) return fail(GRX_ERR_INVALID_ARG, "NULL array pointer");
    if (!(gamma > 1.0)) return fail(GRX_ERR_INVALID_ARG, "gamma must be > 1");
    const cudaError_t e =
        grx::launch_con2prim(cons, metric, p.nc, p.nbox, gamma, prim, nfail, static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return fail_cuda(e, "grx_con2prim launch");
    return GRX_OK;
}

int grx_rk_axpy(const grx_grid* grid, int nghost, double a, const double* x, double b, double dt, const double* rhs,
                double* y, void* cuda_stream) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (const char* why = make_geom(grid, nghost, p)) return fail(GRX_ERR_INVALID_ARG, why);
    if (!x || !rhs || !y) return fail(GRX_ERR_INVALID_ARG, "NULL array pointer");
    const cudaError_t e = grx::launch_rk_axpy(p, a, x, b, dt, rhs, y, static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return fail_cuda(e, "grx_rk_axpy launch");
    return GRX_OK;
}

int grx_valencia_rhs_zrange(const grx_grid* grid, const double* prim, const double* metric, const double* K,
                            const double dx[3], int nghost, int recon, double gamma, double* out, int k_begin, int k_end,
                            void* cuda_stream) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (const char* why = make_geom(grid, nghost, p)) return fail(GRX_ERR_INVALID_ARG, why);
    if (!prim || !metric || !K || !dx || !out) return fail(GRX_ERR_INVALID_ARG, "NULL array pointer");
    if (recon != GRX_RECON_MINMOD && recon != GRX_RECON_MC && recon != GRX_RECON_WENO5)
        return fail(GRX_ERR_INVALID_ARG, "unknown recon");
    if (nghost < (recon == GRX_RECON_WENO5 ? 3 : 2))
        return fail(GRX_ERR_INVALID_ARG, "nghost too small: WENO5 needs 3, minmod/MC need 2 (R29)");
    if (!(gamma > 1.0)) return fail(GRX_ERR_INVALID_ARG, "gamma must be > 1");
    for (int a = 0; a < 3; ++a) {
        if (!(dx[a] > 0.0) || !(1.0 / dx[a] > 0.0)) return fail(GRX_ERR_INVALID_ARG, "dx must be > 0 and finite");
        p.idx[a] = 1.0 / dx[a];
    }
    if (out == prim || out == metric || out == K) return fail(GRX_ERR_INVALID_ARG, "out must not alias an input");
    if (k_begin < 0 || k_end > p.n[2] || k_begin > k_end) return fail(GRX_ERR_INVALID_ARG, "need 0 <= k_begin <= k_end <= nz");
    if (p.nbox != 1 && !(k_begin == 0 && k_end == p.n[2]))
        return fail(GRX_ERR_INVALID_ARG, "a z range of a batch is not contiguous: nbox must be 1");
    if (k_begin == k_end) return GRX_OK;
    p.prim = prim; p.met = metric; p.K = K; p.out = out;
    p.gamma = gamma;
    p.nfallback = t_fallback_counter;
    // the kernel the whole block would get, so that the planes carry the bits of the whole-block call
    const int kernel = choose_kernel(p, recon);
    if (kernel < 0) return fail(GRX_ERR_UNSUPPORTED, "GRX_VARIANT_TMA needs even nx + 2 nghost and 16-byte aligned arrays");
    // the sub-block of planes [k_begin, k_end): same arrays, shifted by k_begin planes, nz = k_end - k_begin; the field
    // stride nc stays that of the whole block
    const int nz_whole = p.n[2];
    const size_t off = (size_t)k_begin * (size_t)p.stride[2];
    p.prim += off; p.met += off; p.K += off; p.out += off;
    p.n[2] = k_end - k_begin;
    p.N[2] = p.n[2] + 2 * p.g;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const cudaError_t e = launch_chosen(kernel, p, recon, st, nz_whole);
    if (e != cudaSuccess) return fail_cuda(e, "grx_valencia_rhs_zrange launch");
    return GRX_OK;
}

int grx_rk_stage(const grx_grid* grid, int nghost, double a, const double* Ua, double b, const double* Ub, double h,
                 const double* L, double* Uout, double* acc, double wdt, const double* metric, double gamma, double* prim,
                 unsigned long long* nfail, void* cuda_stream) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (const char* why = make_geom(grid, nghost, p)) return fail(GRX_ERR_INVALID_ARG, why);
    if (!Ua || !Ub || !L || !Uout || !metric || !prim) return fail(GRX_ERR_INVALID_ARG, "NULL array pointer");
    if (!(gamma > 1.0)) return fail(GRX_ERR_INVALID_ARG, "gamma must be > 1");
    p.met = metric;
    p.gamma = gamma;
    const cudaError_t e = grx::launch_rk_stage(p, a, Ua, b, Ub, h, L, Uout, acc, wdt, prim, nfail,
                                               static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return fail_cuda(e, "grx_rk_stage launch");
    return GRX_OK;
}

int grx_fill_ghosts(const grx_grid* grid, double* prim, int nghost, int bc, int dirs, void* cuda_stream) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (const char* why = make_geom(grid, nghost, p)) return fail(GRX_ERR_INVALID_ARG, why);
    if (!prim) return fail(GRX_ERR_INVALID_ARG, "NULL array pointer");
    if (bc != GRX_BC_COPY && bc != GRX_BC_PERIODIC) return fail(GRX_ERR_INVALID_ARG, "unknown boundary condition");
    if (dirs < 0 || dirs > 7) return fail(GRX_ERR_INVALID_ARG, "dirs is a mask of bits 0..2");
    const cudaError_t e = grx::launch_fill_ghosts(p, prim, bc, dirs, static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return fail_cuda(e, "grx_fill_ghosts launch");
    return GRX_OK;
}

size_t grx_halo_z_bytes(const grx_grid* grid, int nghost) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (make_geom(grid, nghost, p)) return 0;
    return (size_t)p.nbox * 8 * (size_t)p.g * (size_t)p.stride[2] * sizeof(double);
}

int grx_halo_z(const grx_grid* grid, double* prim, int nghost, int side, int unpack, double* buf, void* cuda_stream) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (const char* why = make_geom(grid, nghost, p)) return fail(GRX_ERR_INVALID_ARG, why);
    if (!prim || !buf) return fail(GRX_ERR_INVALID_ARG, "NULL array pointer");
    if (side != 0 && side != 1) return fail(GRX_ERR_INVALID_ARG, "side must be 0 (low) or 1 (high)");
    if (p.n[2] < p.g) return fail(GRX_ERR_INVALID_ARG, "a slab must have at least nghost planes");
    if (p.nbox > 8191) return fail(GRX_ERR_INVALID_ARG, "grx_halo_z takes at most 8191 boxes per call");
    const cudaError_t e = grx::launch_halo_z(p, prim, buf, side, unpack != 0, static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return fail_cuda(e, "grx_halo_z launch");
    return GRX_OK;
}

int grx_valencia_rhs_vertex(const grx_grid* grid, const double* prim, const double* metric_v, const double* K_v,
                            const double dx[3], int nghost, int recon, double gamma, double* out, void* cuda_stream) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (const char* why = make_geom(grid, nghost, p)) return fail(GRX_ERR_INVALID_ARG, why);
    if (!prim || !metric_v || !K_v || !dx || !out) return fail(GRX_ERR_INVALID_ARG, "NULL array pointer");
    if (recon != GRX_RECON_MINMOD && recon != GRX_RECON_MC && recon != GRX_RECON_WENO5)
        return fail(GRX_ERR_INVALID_ARG, "unknown recon");
    if (nghost < (recon == GRX_RECON_WENO5 ? 3 : 2))
        return fail(GRX_ERR_INVALID_ARG, "nghost too small: WENO5 needs 3, minmod/MC need 2 (R29)");
    if (!(gamma > 1.0)) return fail(GRX_ERR_INVALID_ARG, "gamma must be > 1");
    for (int a = 0; a < 3; ++a) {
        if (!(dx[a] > 0.0) || !(1.0 / dx[a] > 0.0)) return fail(GRX_ERR_INVALID_ARG, "dx must be > 0 and finite");
        p.idx[a] = 1.0 / dx[a];
    }
    if (out == prim) return fail(GRX_ERR_INVALID_ARG, "out must not alias an input");
    p.prim = prim; p.met = metric_v; p.K = K_v; p.out = out;
    p.gamma = gamma;
    p.nfallback = t_fallback_counter;
    // the face-once traversal of the LDG kernel with vertex loads; GRX_VARIANT_SIMPLE takes the one-thread-per-cell
    // cross-check traversal (every face evaluated by both of its cells)
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const cudaError_t e = g_variant.load() == GRX_VARIANT_SIMPLE ? grx::launch_rhs_vertex(p, recon, st)
                                                                 : grx::launch_rhs_fused_vertex(p, recon, st);
    if (e != cudaSuccess) return fail_cuda(e, "grx_valencia_rhs_vertex launch");
    return GRX_OK;
}

int grx_tmunu_vertices(const grx_grid* grid, const double* prim, const double* metric_v, int nghost, double gamma, double* T,
                       void* cuda_stream) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (const char* why = make_geom(grid, nghost, p)) return fail(GRX_ERR_INVALID_ARG, why);
    if (!prim || !metric_v || !T) return fail(GRX_ERR_INVALID_ARG, "NULL array pointer");
    if (nghost < 2) return fail(GRX_ERR_INVALID_ARG, "the 4-point interpolation needs 2 ghost cells");
    if (!(gamma > 1.0)) return fail(GRX_ERR_INVALID_ARG, "gamma must be > 1");
    p.prim = prim; p.met = metric_v;
    p.gamma = gamma;
    const cudaError_t e = grx::launch_tmunu_vertex(p, T, static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return fail_cuda(e, "grx_tmunu_vertices launch");
    return GRX_OK;
}

int grx_halo_z_pull(const grx_grid* grid, double* prim, int nghost, const double* below, const double* above, void* cuda_stream) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (const char* why = make_geom(grid, nghost, p)) return fail(GRX_ERR_INVALID_ARG, why);
    if (!prim || !below || !above) return fail(GRX_ERR_INVALID_ARG, "NULL array pointer");
    if (p.n[2] < p.g) return fail(GRX_ERR_INVALID_ARG, "a slab must have at least nghost planes");
    if (p.nbox > 8191) return fail(GRX_ERR_INVALID_ARG, "grx_halo_z_pull takes at most 8191 boxes per call");
    const cudaError_t e = grx::launch_halo_z_pull(p, prim, below, above, static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return fail_cuda(e, "grx_halo_z_pull launch");
    return GRX_OK;
}

size_t grx_ct_workspace_bytes(const grx_grid* grid, int nghost) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (make_geom(grid, nghost, p)) return 0;
    return (size_t)6 * (size_t)p.nc * (size_t)p.nbox * sizeof(double);
}

int grx_valencia_rhs_ct(const grx_grid* grid, const double* prim, const double* metric, const double* K,
                        const double dx[3], int nghost, int recon, double gamma, double* out, void* workspace,
                        size_t workspace_bytes, void* cuda_stream) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (const char* why = make_geom(grid, nghost, p)) return fail(GRX_ERR_INVALID_ARG, why);
    if (!prim || !metric || !K || !dx || !out || !workspace) return fail(GRX_ERR_INVALID_ARG, "NULL array pointer");
    if (recon != GRX_RECON_MINMOD && recon != GRX_RECON_MC && recon != GRX_RECON_WENO5)
        return fail(GRX_ERR_INVALID_ARG, "unknown recon");
    if (nghost < (recon == GRX_RECON_WENO5 ? 3 : 2))
        return fail(GRX_ERR_INVALID_ARG, "nghost too small: WENO5 needs 3, minmod/MC need 2 (R29)");
    if (!(gamma > 1.0)) return fail(GRX_ERR_INVALID_ARG, "gamma must be > 1");
    for (int a = 0; a < 3; ++a) {
        if (!(dx[a] > 0.0) || !(1.0 / dx[a] > 0.0)) return fail(GRX_ERR_INVALID_ARG, "dx must be > 0 and finite");
        p.idx[a] = 1.0 / dx[a];
    }
    if (out == prim || out == metric || out == K) return fail(GRX_ERR_INVALID_ARG, "out must not alias an input");
    if (workspace_bytes < (size_t)6 * (size_t)p.nc * (size_t)p.nbox * sizeof(double))
        return fail(GRX_ERR_INVALID_ARG, "workspace too small");
    p.prim = prim; p.met = metric; p.K = K; p.out = out;
    p.gamma = gamma;
    p.nfallback = t_fallback_counter;
    p.fb = static_cast<double*>(workspace);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    bool unsupported = false;
    const cudaError_t e = launch_rhs_ct(p, recon, st, &unsupported);
    if (unsupported) return fail(GRX_ERR_UNSUPPORTED, "GRX_VARIANT_TMA needs even nx + 2 nghost and 16-byte aligned arrays");
    if (e != cudaSuccess) return fail_cuda(e, "grx_valencia_rhs_ct launch");
    return GRX_OK;
}

size_t grx_ct_static_max_bytes(void) { return GRX_CT_STATIC_MAX_BYTES; }

// Same checks and the same launch sequence as grx_valencia_rhs_ct; the six face-flux arrays go to the library's own fixed
// device array instead of a caller's workspace.  No allocation on any call.  The array is shared by every call on the
// device: calls that overlap on the GPU race (include/grx.h).  Nothing is cleared: launch_rhs_ct writes every face flux
// the curl kernel reads before that kernel runs, whatever an earlier call left behind.
int grx_valencia_rhs_ct_static(const grx_grid* grid, const double* prim, const double* metric, const double* K,
                               const double dx[3], int nghost, int recon, double gamma, double* out, void* cuda_stream) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (const char* why = make_geom(grid, nghost, p)) return fail(GRX_ERR_INVALID_ARG, why);
    if (!prim || !metric || !K || !dx || !out) return fail(GRX_ERR_INVALID_ARG, "NULL array pointer");
    if (recon != GRX_RECON_MINMOD && recon != GRX_RECON_MC && recon != GRX_RECON_WENO5)
        return fail(GRX_ERR_INVALID_ARG, "unknown recon");
    if (nghost < (recon == GRX_RECON_WENO5 ? 3 : 2))
        return fail(GRX_ERR_INVALID_ARG, "nghost too small: WENO5 needs 3, minmod/MC need 2 (R29)");
    if (!(gamma > 1.0)) return fail(GRX_ERR_INVALID_ARG, "gamma must be > 1");
    for (int a = 0; a < 3; ++a) {
        if (!(dx[a] > 0.0) || !(1.0 / dx[a] > 0.0)) return fail(GRX_ERR_INVALID_ARG, "dx must be > 0 and finite");
        p.idx[a] = 1.0 / dx[a];
    }
    if (out == prim || out == metric || out == K) return fail(GRX_ERR_INVALID_ARG, "out must not alias an input");
    const unsigned long long need = 6ULL * (unsigned long long)p.nc * (unsigned long long)p.nbox;   // <= 6 * 2^31 * 2^16
    if (need > CT_STATIC_DOUBLES) {
        std::snprintf(t_err, sizeof(t_err),
                      "the call needs %llu bytes of face fluxes, which exceeds the static scratch of %llu bytes "
                      "(GRX_CT_STATIC_MAX_BYTES): split the call or use grx_valencia_rhs_ct with a workspace",
                      need * 8ULL, (unsigned long long)GRX_CT_STATIC_MAX_BYTES);
        return GRX_ERR_INVALID_ARG;
    }
    double* scratch = nullptr;
    cudaError_t e = ct_static_scratch(&scratch);
    if (e != cudaSuccess) return fail_cuda(e, "grx_valencia_rhs_ct_static: address of the static scratch");
    p.prim = prim; p.met = metric; p.K = K; p.out = out;
    p.gamma = gamma;
    p.nfallback = t_fallback_counter;
    p.fb = scratch;
    bool unsupported = false;
    e = launch_rhs_ct(p, recon, static_cast<cudaStream_t>(cuda_stream), &unsupported);
    if (unsupported) return fail(GRX_ERR_UNSUPPORTED, "GRX_VARIANT_TMA needs even nx + 2 nghost and 16-byte aligned arrays");
    if (e != cudaSuccess) return fail_cuda(e, "grx_valencia_rhs_ct_static launch");
    return GRX_OK;
}

size_t grx_step_workspace_bytes(const grx_grid* grid, int nghost, int rk_order) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (make_geom(grid, nghost, p) || (rk_order != 2 && rk_order != 4)) return 0;
    return (size_t)(rk_order == 2 ? 2 : 3) * 8 * (size_t)p.nc * (size_t)p.nbox * sizeof(double);
}

size_t grx_step_ct_workspace_bytes(const grx_grid* grid, int nghost, int rk_order) {
    const size_t a = grx_step_workspace_bytes(grid, nghost, rk_order), b = grx_ct_workspace_bytes(grid, nghost);
    return (a && b) ? a + b : 0;
}

static int step_rk_impl(const grx_grid* grid, double* cons, double* prim, const double* metric, const double* K,
                        const double dx[3], int nghost, int recon, double gamma, double dt, int rk_order, int bc, int nsteps,
                        void* workspace, size_t workspace_bytes, unsigned long long* nfail, void* cuda_stream, bool ct);

int grx_step_rk(const grx_grid* grid, double* cons, double* prim, const double* metric, const double* K,
                const double dx[3], int nghost, int recon, double gamma, double dt, int rk_order, int bc, int nsteps,
                void* workspace, size_t workspace_bytes, unsigned long long* nfail, void* cuda_stream) {
    return step_rk_impl(grid, cons, prim, metric, K, dx, nghost, recon, gamma, dt, rk_order, bc, nsteps, workspace,
                        workspace_bytes, nfail, cuda_stream, false);
}

int grx_step_rk_ct(const grx_grid* grid, double* cons, double* prim, const double* metric, const double* K,
                   const double dx[3], int nghost, int recon, double gamma, double dt, int rk_order, int bc, int nsteps,
                   void* workspace, size_t workspace_bytes, unsigned long long* nfail, void* cuda_stream) {
    return step_rk_impl(grid, cons, prim, metric, K, dx, nghost, recon, gamma, dt, rk_order, bc, nsteps, workspace,
                        workspace_bytes, nfail, cuda_stream, true);
}

static int step_rk_impl(const grx_grid* grid, double* cons, double* prim, const double* metric, const double* K,
                        const double dx[3], int nghost, int recon, double gamma, double dt, int rk_order, int bc, int nsteps,
                        void* workspace, size_t workspace_bytes, unsigned long long* nfail, void* cuda_stream, bool ct) {
    grx::RhsParams p;
    std::memset(&p, 0, sizeof(p));
    if (const char* why = make_geom(grid, nghost, p)) return fail(GRX_ERR_INVALID_ARG, why);
    if (!cons || !prim || !metric || !K || !dx || !workspace) return fail(GRX_ERR_INVALID_ARG, "NULL array pointer");
    if (recon != GRX_RECON_MINMOD && recon != GRX_RECON_MC && recon != GRX_RECON_WENO5)
        return fail(GRX_ERR_INVALID_ARG, "unknown recon");
    if (nghost < (recon == GRX_RECON_WENO5 ? 3 : 2))
        return fail(GRX_ERR_INVALID_ARG, "nghost too small: WENO5 needs 3, minmod/MC need 2 (R29)");
    if (!(gamma > 1.0)) return fail(GRX_ERR_INVALID_ARG, "gamma must be > 1");
    if (rk_order != 2 && rk_order != 4) return fail(GRX_ERR_INVALID_ARG, "rk_order must be 2 or 4");
    if (bc != GRX_BC_COPY && bc != GRX_BC_PERIODIC) return fail(GRX_ERR_INVALID_ARG, "unknown boundary condition");
    if (nsteps < 0 || !(dt == dt)) return fail(GRX_ERR_INVALID_ARG, "nsteps must be >= 0 and dt a number");
    for (int a = 0; a < 3; ++a) {
        if (!(dx[a] > 0.0) || !(1.0 / dx[a] > 0.0)) return fail(GRX_ERR_INVALID_ARG, "dx must be > 0 and finite");
        p.idx[a] = 1.0 / dx[a];
    }
    const size_t arr = 8 * (size_t)p.nc * (size_t)p.nbox;
    const size_t nrk = (size_t)(rk_order == 2 ? 2 : 3);
    if (workspace_bytes < (nrk * arr + (ct ? 6 * (size_t)p.nc * (size_t)p.nbox : 0)) * sizeof(double))
        return fail(GRX_ERR_INVALID_ARG, "workspace too small");
    double* U0 = static_cast<double*>(workspace);
    double* L = U0 + arr;
    double* acc = rk_order == 4 ? L + arr : nullptr;
    p.prim = prim; p.met = metric; p.K = K; p.out = L;
    p.gamma = gamma;
    p.nfallback = nullptr;
    p.fb = ct ? U0 + nrk * arr : nullptr;      // the six face-flux arrays of constrained transport follow the RK arrays
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    cudaError_t e = cudaSuccess;
    auto rhs = [&]() { return ct ? launch_rhs_ct(p, recon, st, nullptr) : launch_variant(p, recon, st); };
    auto stage = [&](double a, const double* Ua, double b, const double* Ub, double h, double* Uout, double* ac, double wdt) {
        cudaError_t r = grx::launch_rk_stage(p, a, Ua, b, Ub, h, L, Uout, ac, wdt, prim, nfail, st);
        return r != cudaSuccess ? r : grx::launch_fill_ghosts(p, prim, bc, 7, st);
    };
    // `cons` keeps U^n until the last stage of a step overwrites it; the intermediate stage states go to the first
    // workspace array (W) -- no copy of cons per step.  The next right-hand side reads prim only, so W is needed again
    // only where a stage combines it (RK2).  L and W live in the workspace: their ghost cells are never read or written.
    double* W = U0;
    for (int s = 0; s < nsteps && e == cudaSuccess; ++s) {
        if (rk_order == 2) {
            e = rhs();
            if (e == cudaSuccess) e = stage(0.0, cons, 1.0, cons, dt, W, nullptr, 0.0);      // U1 = U0 + dt L(P0)
            if (e == cudaSuccess) e = rhs();
            if (e == cudaSuccess) e = stage(0.5, cons, 0.5, W, dt, cons, nullptr, 0.0);      // U = 1/2 U0 + 1/2 (U1 + dt L(P1))
        } else {
            const double w[4] = {1.0 / 6.0, 1.0 / 3.0, 1.0 / 3.0, 1.0 / 6.0}, hs[3] = {0.5, 0.5, 1.0};
            e = cudaMemcpyAsync(acc, cons, arr * sizeof(double), cudaMemcpyDeviceToDevice, st);
            for (int k = 0; k < 3 && e == cudaSuccess; ++k) {
                e = rhs();
                if (e == cudaSuccess) e = stage(0.0, cons, 1.0, cons, hs[k] * dt, W, acc, w[k] * dt);   // U = U0 + h dt k_k
            }
            if (e == cudaSuccess) e = rhs();
            // the last weight goes in as the stage's own step: U = (U0 + dt/6 (k1 + 2 k2 + 2 k3)) + dt/6 k4
            if (e == cudaSuccess) e = stage(0.0, cons, 1.0, acc, w[3] * dt, cons, nullptr, 0.0);        // U = acc + dt/6 k4
        }
    }
    if (e != cudaSuccess) return fail_cuda(e, "grx_step_rk");
    return GRX_OK;
}

int grx_debug_set_fallback_counter(unsigned long long* counter) {
    t_fallback_counter = counter;
    return GRX_OK;
}

int grx_debug_fallback_count(unsigned long long* host_out, void* cuda_stream) {
    if (!host_out) return fail(GRX_ERR_INVALID_ARG, "host_out is NULL");
    if (!t_fallback_counter)
        return fail(GRX_ERR_INVALID_ARG, "no fallback counter registered on this thread (grx_debug_set_fallback_counter)");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    cudaError_t e = cudaMemcpyAsync(host_out, t_fallback_counter, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return fail_cuda(e, "grx_debug_fallback_count");
    return GRX_OK;
}

int grx_set_variant(int variant) {
    if (variant != GRX_VARIANT_AUTO && variant != GRX_VARIANT_SIMPLE && variant != GRX_VARIANT_LDG && variant != GRX_VARIANT_TMA)
        return fail(GRX_ERR_INVALID_ARG, "unknown variant");
    g_variant.store(variant);
    return GRX_OK;
}

int grx_selftest_math(const double* x, double* y, size_t n, void* cuda_stream) {
    if (n && (!x || !y)) return fail(GRX_ERR_INVALID_ARG, "NULL array pointer");
    const cudaError_t e = grx::launch_selftest_math(x, y, n, static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return fail_cuda(e, "grx_selftest_math launch");
    return GRX_OK;
}

const char* grx_last_error(void) { return t_err; }
int grx_version(void) { return 100; }   /* 0.1.0 */
double grx_weno_eps(void) { return grx::WENO_EPS; }
double grx_v2max(void) { return grx::V2MAX; }

}  // extern "C"

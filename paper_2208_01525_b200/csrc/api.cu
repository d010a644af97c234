// api.cu -- the C ABI of libu1u1.so (include/u1u1.h): context, host-side per-step scalars
// (PAPER.md:133 Eq. 19, :147 Eq. 22, :89 Eq. 12), launch sequencing, derived diagnostics
// (Eq. 31-37).  No device memory is allocated here; no CPU compute path exists.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>

#include "../../include/u1u1.h"
#include "../../include/u1u1_tuning.h"
#include "common.cuh"
#include "kernels.h"
#include "stage.cuh"

using namespace u1u1;

struct u1u1_ctx {
    float *state = nullptr;      // caller-owned: [pos0 | pos1 | mom]
    size_t state_bytes = 0;
    uint8_t *scratch = nullptr;  // caller-owned
    size_t scratch_bytes = 0;
    cudaStream_t stream = nullptr;
    int N = 0;
    size_t V = 0;                // sites in one buffer (N^3; N * N * (nz_own + 2) for a z slab)
    // z slab of a lattice split over several GPUs (u1u1_configure_slab; 0 = ordinary cubic lattice)
    int nz_own = 0;
    int64_t z_first = 0;         // global index of the slab's first own plane
    float *peer_up = nullptr, *peer_dn = nullptr;   // state buffers of the slabs above / below
    double dx = 0;
    u1u1_params prm{};
    bool configured = false;
    int cur = 0;                 // which ping-pong buffer holds the current positions
    // time bookkeeping for the diagnostic weights
    double tau_pos = 0.0;        // conformal time of the positions
    double a = 1.0, c = 1.0, cG = 1.0;
    bool diag_valid = false;     // scratch holds the cell arrays of the current state
    bool codes_valid = false;    // scratch holds the winding codes of the current state
    bool labels_valid = false;   // scratch holds segment labels of the current state
    uint64_t launches = 0;
    uint32_t tuning = 0;         // experimental switches (u1u1_set_tuning, include/u1u1_tuning.h)
    double last_max_theta = 0.0; // of the last diagnostics sweep since configure (range_reduce = 2)
    // device properties and TMA tensor maps, set up on the first launch (nothing here needs a GPU before that)
    int sms = 0;
    bool maps_ready = false;
    PackMaps pos_halo[2], mom_halo[2], mom_tile[2];     // momenta: [0] the buffer inside `state`, [1] the aux buffer
    PackMaps mom_tile_tb[2];                             // tile boxes of the two-steps-per-pass kernel's tile
    PackMaps pos_halo2[2];                               // two-site-halo boxes of the positions (two-steps-per-pass kernel)
    // optional second momentum buffer (u1u1_set_aux): enables the two-steps-per-pass kernel, which reads the momenta
    // from one buffer and writes them to the other
    float *aux = nullptr;
    size_t aux_bytes = 0;
    int mcur = 0;                // which momentum buffer is current: 0 = inside `state`, 1 = aux
    // second stream and events of the pipelined host copies, created on first use
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_kernel[2] = {nullptr, nullptr}, ev_copy[2] = {nullptr, nullptr};
    std::string err;
};

static thread_local std::string g_create_err;   // message of a failed u1u1_create on this thread

static int fail(u1u1_ctx *ctx, int code, const std::string &msg)
{
    if (ctx) ctx->err = msg; else g_create_err = msg;
    return code;
}

static int cuda_fail(u1u1_ctx *ctx, cudaError_t e, const char *where)
{
    return fail(ctx, U1U1_ECUDA, std::string(where) + ": " + cudaGetErrorString(e));
}

static bool size_ok(int32_t N) { return N >= 8 && N <= 1024 && (N % 4) == 0; }

// scratch layout: [cells 2V][work 8V] pad-> [partials RED_MAX_BLOCKS*RED_SLOTS doubles][result 64 doubles]
// work = winding codes 6V (export_windings) | segment labels 4V + sizes 4V (pq_segments) | two staging planes 4V + 4V
// (host copies): the cell arrays survive all of them.
static size_t scratch_partials_offset(size_t V) { return ((10 * V + 255) / 256) * 256; }

extern "C" size_t u1u1_state_bytes(int32_t N)
{
    if (!size_ok(N)) return 0;
    return (size_t)(2 * NPOS + NMOM) * (size_t)N * N * N * sizeof(float);
}

extern "C" size_t u1u1_scratch_bytes(int32_t N)
{
    if (!size_ok(N)) return 0;
    const size_t V = (size_t)N * N * N;
    return scratch_partials_offset(V) + ((size_t)RED_MAX_BLOCKS * RED_SLOTS + 64) * sizeof(double);
}

extern "C" size_t u1u1_aux_bytes(int32_t N)
{
    if (!size_ok(N)) return 0;
    return (size_t)NMOM * (size_t)N * N * N * sizeof(float);
}

extern "C" int u1u1_set_aux(u1u1_ctx *ctx, void *aux_dev, size_t aux_bytes)
{
    if (!ctx) return U1U1_EINVAL;
    if (ctx->nz_own) return fail(ctx, U1U1_ESTATE, "set_aux is not available on a z slab");
    if (aux_dev && (((uintptr_t)aux_dev & 255) || (ctx->configured && aux_bytes < u1u1_aux_bytes(ctx->N))))
        return fail(ctx, U1U1_ESIZE, "aux buffer must be 256-byte aligned and hold u1u1_aux_bytes(N)");
    if (ctx->mcur == 1) {                     // the momenta live in the old aux buffer: bring them home first
        cudaError_t e = cudaMemcpyAsync(ctx->state + (size_t)2 * NPOS * ctx->V, ctx->aux, (size_t)NMOM * ctx->V * sizeof(float),
                                        cudaMemcpyDeviceToDevice, ctx->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "set_aux: moving the momenta back");
        ctx->mcur = 0;
    }
    ctx->aux = (float *)aux_dev;
    ctx->aux_bytes = aux_dev ? aux_bytes : 0;
    ctx->maps_ready = false;
    return U1U1_OK;
}

extern "C" int u1u1_create(u1u1_ctx **out, void *state_dev, size_t state_bytes, void *scratch_dev,
                           size_t scratch_bytes, void *cuda_stream)
{
    if (!out || !state_dev || !scratch_dev) return fail(nullptr, U1U1_EINVAL, "u1u1_create: NULL argument");
    if (((uintptr_t)state_dev & 255) || ((uintptr_t)scratch_dev & 255))
        return fail(nullptr, U1U1_EINVAL, "u1u1_create: device buffers must be 256-byte aligned");
    u1u1_ctx *ctx = new (std::nothrow) u1u1_ctx;
    if (!ctx) return fail(nullptr, U1U1_EINVAL, "u1u1_create: out of host memory");
    ctx->state = (float *)state_dev;
    ctx->state_bytes = state_bytes;
    ctx->scratch = (uint8_t *)scratch_dev;
    ctx->scratch_bytes = scratch_bytes;
    ctx->stream = (cudaStream_t)cuda_stream;
    *out = ctx;
    return U1U1_OK;
}

extern "C" void u1u1_destroy(u1u1_ctx *ctx)
{
    if (!ctx) return;
    for (int b = 0; b < 2; b++) {
        if (ctx->ev_kernel[b]) cudaEventDestroy(ctx->ev_kernel[b]);
        if (ctx->ev_copy[b]) cudaEventDestroy(ctx->ev_copy[b]);
    }
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    delete ctx;
}

extern "C" const char *u1u1_last_error(const u1u1_ctx *ctx)
{
    return ctx ? ctx->err.c_str() : g_create_err.c_str();
}

extern "C" uint64_t u1u1_launch_count(const u1u1_ctx *ctx) { return ctx ? ctx->launches : 0; }

static int check_params(u1u1_ctx *ctx, const u1u1_params *p)
{
    if (!p) return fail(ctx, U1U1_EINVAL, "params is NULL");
    if (p->struct_size != sizeof(u1u1_params))
        return fail(ctx, U1U1_EINVAL, "params->struct_size does not match this library's u1u1_params");
    if (!(p->lambda1 > 0 && p->lambda2 > 0 && p->e1 > 0 && p->e2 > 0 && p->eta1 > 0 && p->eta2 > 0))
        return fail(ctx, U1U1_EPARAM, "couplings and symmetry-breaking scales must be positive");
    if (!(p->kappa >= 0 && p->kappa < 0.5 * std::sqrt(p->lambda1 * p->lambda2)))
        return fail(ctx, U1U1_EPARAM, "need 0 <= kappa < sqrt(lambda1 lambda2)/2 (PAPER.md:55)");
    if (!(p->dtau > 0) || !(p->tau_norm > 0) || !(p->friction > 0 && p->friction <= 1.0))
        return fail(ctx, U1U1_EPARAM, "need dtau > 0, tau_norm > 0, 0 < friction <= 1");
    if (p->init_kind != 0 && p->init_kind != 1) return fail(ctx, U1U1_EINVAL, "init_kind must be 0 or 1");
    if (p->init_kind == 1 && (!(p->smooth_width > 0) || p->smooth_trunc < 1 || p->smooth_trunc > 32))
        return fail(ctx, U1U1_EINVAL, "init_kind 1 needs smooth_width > 0 and 1 <= smooth_trunc <= 32");
    if (p->kernel_variant < 0 || p->kernel_variant > 7) return fail(ctx, U1U1_EINVAL, "kernel_variant must be 0..7");
    if (p->range_reduce < 0 || p->range_reduce > 2 || p->reserved != 0)
        return fail(ctx, U1U1_EINVAL, "range_reduce must be 0 (off), 1 (on) or 2 (automatic), reserved 0");
    return U1U1_OK;
}

// switches handed to the kernels: the experimental mask + 2048 when the range reduction of the link phases is on
static int kernel_flags(const u1u1_ctx *ctx)
{
    const int rr = ctx->prm.range_reduce;
    const bool reduce = rr == 1 || (rr == 2 && ctx->last_max_theta > 10.0);
    return (int)ctx->tuning | (reduce ? 2048 : 0);
}

extern "C" int u1u1_set_tuning(u1u1_ctx *ctx, uint32_t flags)
{
    if (!ctx) return U1U1_EINVAL;
    if (flags & ~U1U1_TUNE_ALL) return fail(ctx, U1U1_EINVAL, "set_tuning: unknown switch (see include/u1u1_tuning.h)");
    ctx->tuning = flags;
    return U1U1_OK;
}

static float *pos_buf(u1u1_ctx *ctx, int which) { return ctx->state + (size_t)which * NPOS * ctx->V; }
static float *mom_buf_at(u1u1_ctx *ctx, int which) { return which ? ctx->aux : ctx->state + (size_t)2 * NPOS * ctx->V; }
static float *mom_buf(u1u1_ctx *ctx) { return mom_buf_at(ctx, ctx->mcur); }
static uint8_t *cells_buf(u1u1_ctx *ctx) { return ctx->scratch; }
static uint8_t *work_buf(u1u1_ctx *ctx) { return ctx->scratch + 2 * ctx->V; }
static double *partials(u1u1_ctx *ctx) { return (double *)(ctx->scratch + scratch_partials_offset(ctx->V)); }
static double *result(u1u1_ctx *ctx) { return partials(ctx) + (size_t)RED_MAX_BLOCKS * RED_SLOTS; }

// SM count of the current device and the tensor maps of this context's buffers, once per configure
static int prepare_device(u1u1_ctx *ctx)
{
    if (!ctx->sms) {
        int dev = 0, sms = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess || sms < 1) return cuda_fail(ctx, e, "querying the SM count");
        ctx->sms = sms;
    }
    if (!ctx->maps_ready && step_tiled_uses_tma(ctx->N)) {
        const int NZ = ctx->nz_own ? ctx->nz_own + 2 : ctx->N;
        bool ok = encode_halo_maps(&ctx->pos_halo[0], pos_buf(ctx, 0), ctx->V, ctx->N, NZ) &&
                        encode_halo_maps(&ctx->pos_halo[1], pos_buf(ctx, 1), ctx->V, ctx->N, NZ) &&
                        encode_halo_maps(&ctx->mom_halo[0], mom_buf_at(ctx, 0), ctx->V, ctx->N, NZ) &&
                        encode_tile_maps(&ctx->mom_tile[0], mom_buf_at(ctx, 0), ctx->V, ctx->N, NZ);
        if (ok && ctx->aux)
            ok = encode_halo_maps(&ctx->mom_halo[1], ctx->aux, ctx->V, ctx->N, NZ) &&
                 encode_tile_maps(&ctx->mom_tile[1], ctx->aux, ctx->V, ctx->N, NZ) &&
                 encode_tb_tile_maps(&ctx->mom_tile_tb[0], mom_buf_at(ctx, 0), ctx->V, ctx->N, NZ) &&
                 encode_tb_tile_maps(&ctx->mom_tile_tb[1], ctx->aux, ctx->V, ctx->N, NZ) &&
                 encode_halo2_maps(&ctx->pos_halo2[0], pos_buf(ctx, 0), ctx->V, ctx->N, NZ) &&
                 encode_halo2_maps(&ctx->pos_halo2[1], pos_buf(ctx, 1), ctx->V, ctx->N, NZ);
        if (!ok) return fail(ctx, U1U1_ECUDA, "cuTensorMapEncodeTiled unavailable or rejected the layout (TMA is required)");
        ctx->maps_ready = true;
    }
    return U1U1_OK;
}

extern "C" int u1u1_configure(u1u1_ctx *ctx, int32_t N, double dx, const u1u1_params *params)
{
    if (!ctx) return U1U1_EINVAL;
    if (!size_ok(N)) return fail(ctx, U1U1_ESIZE, "N must be a multiple of 4 with 8 <= N <= 1024");
    if (!(dx > 0)) return fail(ctx, U1U1_EINVAL, "dx must be positive");
    if (int rc = check_params(ctx, params)) return rc;
    if (ctx->state_bytes < u1u1_state_bytes(N)) return fail(ctx, U1U1_ESIZE, "state buffer smaller than u1u1_state_bytes(N)");
    if (ctx->scratch_bytes < u1u1_scratch_bytes(N)) return fail(ctx, U1U1_ESIZE, "scratch buffer smaller than u1u1_scratch_bytes(N)");
    if (ctx->aux && ctx->aux_bytes < u1u1_aux_bytes(N)) return fail(ctx, U1U1_ESIZE, "aux buffer smaller than u1u1_aux_bytes(N)");
    ctx->N = N;
    ctx->V = (size_t)N * N * N;
    ctx->nz_own = 0;
    ctx->z_first = 0;
    ctx->peer_up = ctx->peer_dn = nullptr;
    ctx->dx = dx;
    ctx->prm = *params;
    ctx->configured = true;
    ctx->cur = 0;
    ctx->mcur = 0;
    ctx->tau_pos = params->tau_norm;
    ctx->a = ctx->c = ctx->cG = 1.0;
    ctx->diag_valid = ctx->codes_valid = ctx->labels_valid = false;
    ctx->maps_ready = false;
    ctx->last_max_theta = 0.0;
    return U1U1_OK;
}

extern "C" int u1u1_set_params(u1u1_ctx *ctx, const u1u1_params *params)
{
    if (!ctx) return U1U1_EINVAL;
    if (!ctx->configured) return fail(ctx, U1U1_ESTATE, "set_params before configure/init_fields");
    if (int rc = check_params(ctx, params)) return rc;
    ctx->prm = *params;
    return U1U1_OK;
}

extern "C" int u1u1_init_fields(u1u1_ctx *ctx, uint64_t seed, int32_t N, double dx, const u1u1_params *params)
{
    if (int rc = u1u1_configure(ctx, N, dx, params)) return rc;
    const size_t V = ctx->V;
    cudaError_t e = cudaMemsetAsync(ctx->state, 0, u1u1_state_bytes(N), ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "init_fields memset");
    if (params->init_kind == 0) {
        e = launch_init_random_phase(pos_buf(ctx, 0), V, 0, 0, seed, params->eta1, params->eta2, ctx->stream);
        ctx->launches += 1;
    } else {
        // the second position buffer and the momentum buffer (adjacent: 80 B/site) are free at init time: two fp64
        // temporaries of 4 planes each (64 B/site)
        double *tmp = (double *)pos_buf(ctx, 1);
        e = launch_init_smoothed(pos_buf(ctx, 0), tmp, tmp + 4 * V, V, N, seed, params->smooth_width,
                                 params->smooth_trunc, params->eta1, params->eta2, ctx->stream);
        ctx->launches += 5;
        if (e == cudaSuccess) e = cudaMemsetAsync(tmp, 0, (size_t)(NPOS + NMOM) * V * sizeof(float), ctx->stream);
    }
    if (e != cudaSuccess) return cuda_fail(ctx, e, "init_fields");
    return U1U1_OK;
}

// a, c = a^{2s}, delta, omega at conformal time tau (fp64).
static void scalars_at(const u1u1_ctx *ctx, double tau, double m, double s, double &a, double &c,
                       double &delta, double &omega)
{
    const double p = m / (1.0 - m);
    a = (m == 0.0) ? 1.0 : std::pow(tau / ctx->prm.tau_norm, p);
    c = std::pow(a, 2.0 * s);
    delta = (m == 0.0) ? 0.0 : p * ctx->prm.dtau / tau;   // (1/2) alpha (dln a/dln tau) dtau/tau, alpha = 2
    omega = delta * (1.0 - s);
}

extern "C" int u1u1_set_time(u1u1_ctx *ctx, double tau, double era_m, double s)
{
    if (!ctx) return U1U1_EINVAL;
    if (!ctx->configured) return fail(ctx, U1U1_ESTATE, "set_time before configure/init_fields");
    if (!(era_m >= 0 && era_m < 1) || !(tau > 0 || era_m == 0)) return fail(ctx, U1U1_EINVAL, "need 0 <= era_m < 1 and tau > 0");
    double delta, omega;
    scalars_at(ctx, tau, era_m, s, ctx->a, ctx->c, delta, omega);
    ctx->cG = ctx->c;
    ctx->tau_pos = tau;
    return U1U1_OK;
}

// kernel_variant (low 4 bits, include/u1u1.h) -> template instance of the tiled kernel; -1 = reference kernel
static int tiled_mode(int kv)
{
    static const int mode_of[8] = {5, -1, 3, -1, 1, 2, 0, 4};
    return mode_of[kv & 7];
}

static cudaError_t launch_step(u1u1_ctx *ctx, const StepCoef &q)
{
    const int kv = ctx->prm.kernel_variant & 15;
    Lattice L{};
    L.pos_in = pos_buf(ctx, ctx->cur);
    L.pos_out = pos_buf(ctx, ctx->cur ^ 1);
    L.mom = mom_buf(ctx);
    L.V = ctx->V;
    L.N = ctx->N;
    if (ctx->nz_own) {                       // z slab: neighbours have the same shape, their pos_out is the same ping-pong index
        L.nz_own = ctx->nz_own;
        L.peer_up_out = ctx->peer_up + (size_t)(ctx->cur ^ 1) * NPOS * ctx->V;
        L.peer_dn_out = ctx->peer_dn + (size_t)(ctx->cur ^ 1) * NPOS * ctx->V;
        L.peer_dn_plane = (size_t)ctx->nz_own + 1;
        L.peer_up_V = L.peer_dn_V = ctx->V;
    }
    const bool tiled = tiled_mode(kv) >= 0 && step_tiled_supports(ctx->N);
    if (!tiled) return launch_step_ref(L, q, ctx->stream, kv == 3);
    StepMaps maps;
    if (ctx->maps_ready) {
        maps.pos = ctx->pos_halo[ctx->cur];
        maps.mom = ctx->mom_tile[ctx->mcur];
    }
    return launch_step_tiled(L, q, ctx->stream, tiled_mode(kv), ctx->maps_ready ? &maps : nullptr, ctx->sms);
}

// Two steps per pass (step_tb.cu) whenever the caller has provided the second momentum buffer (u1u1_set_aux): default
// kernel variant, cubic lattice; tuning flags 1 (scalar chain) and 256 keep the one-step kernel.
static bool pairs_enabled(const u1u1_ctx *ctx)
{
    return ctx->aux && !ctx->nz_own && ctx->prm.kernel_variant == 0 && !(ctx->tuning & (1 | 256)) && step_tb_supports(ctx->N);
}

// one launch, two steps: positions to the other ping-pong buffer, momenta from the current to the other momentum buffer
static cudaError_t launch_two_steps(u1u1_ctx *ctx, const StepCoef &q1, const StepCoef &q2)
{
    TbLattice L{pos_buf(ctx, ctx->cur), pos_buf(ctx, ctx->cur ^ 1), mom_buf_at(ctx, ctx->mcur), mom_buf_at(ctx, ctx->mcur ^ 1),
                ctx->V, ctx->N};
    TbMaps maps;
    if (ctx->maps_ready) {
        maps.pos = ctx->pos_halo2[ctx->cur];
        maps.mom = ctx->mom_tile_tb[ctx->mcur];
    }
    cudaError_t e = launch_step_tb(L, q1, q2, ctx->stream, ctx->maps_ready ? &maps : nullptr, ctx->sms);
    ctx->mcur ^= 1;
    ctx->cur ^= 1;
    return e;
}

// calls that read z neighbours through the periodic wrap of a cubic buffer are not available on a z slab
static int cubic_only(u1u1_ctx *ctx, const char *what)
{
    if (!ctx->nz_own) return U1U1_OK;
    return fail(ctx, U1U1_ESTATE, std::string(what) + " is not available on a z slab (u1u1_configure_slab)");
}

static void invalidate(u1u1_ctx *ctx) { ctx->diag_valid = ctx->codes_valid = ctx->labels_valid = false; }

extern "C" int u1u1_step(u1u1_ctx *ctx, int32_t n, double tau, double era_m, double s)
{
    if (!ctx) return U1U1_EINVAL;
    if (!ctx->configured) return fail(ctx, U1U1_ESTATE, "step before configure/init_fields");
    if (n < 0) return fail(ctx, U1U1_EINVAL, "n must be >= 0");
    if (!(era_m >= 0 && era_m < 1)) return fail(ctx, U1U1_EINVAL, "era_m must satisfy 0 <= m < 1");
    if (era_m != 0 && !(tau > 0)) return fail(ctx, U1U1_EINVAL, "tau must be positive in an expanding background");
    if (ctx->nz_own && (!ctx->peer_up || !ctx->peer_dn)) return fail(ctx, U1U1_ESTATE, "step on a z slab needs u1u1_set_slab_peers first");
    if (ctx->nz_own && (n > 1 || (ctx->prm.kernel_variant & 15) != 0))
        return fail(ctx, U1U1_EINVAL, "a z slab steps one step per call (the ranks synchronise in between) with kernel_variant 0");
    const u1u1_params &P = ctx->prm;
    const double dx = ctx->dx, dt = P.dtau, f = P.friction;
    // coefficients of the step that starts at conformal time tk (fp64 on the host, rounded once)
    auto coef_at = [&](double tk, StepCoef &q, double &c, double &delta, double &omega) -> int {
        double a;
        scalars_at(ctx, tk, era_m, s, a, c, delta, omega);
        const double lam = std::fmax(P.lambda1 * P.eta1 * P.eta1, P.lambda2 * P.eta2 * P.eta2) +
                           2.0 * P.kappa * std::fmax(P.eta1 * P.eta1, P.eta2 * P.eta2);
        if (dt * dt * (12.0 / (dx * dx) + lam * c) >= 4.0) {
            char buf[160];
            snprintf(buf, sizeof buf, "leapfrog unstable at tau=%g: dtau^2 (12/dx^2 + (lambda+2kappa) sigma^2 a^{2s}) >= 4 (a^{2s}=%g)", tk, c);
            return fail(ctx, U1U1_EUNSTABLE, buf);
        }
        q.aS = (float)(f * (1.0 - delta) / (1.0 + delta));
        q.bS = (float)(f * dt / (1.0 + delta));
        q.aG = (float)(f * (1.0 - omega) / (1.0 + omega));
        q.bG = (float)(f * dt / (1.0 + omega));
        q.lamh1 = (float)(0.5 * P.lambda1 * c);
        q.lamh2 = (float)(0.5 * P.lambda2 * c);
        q.kap = (float)(P.kappa * c);
        q.sig1sq = (float)(P.eta1 * P.eta1);
        q.sig2sq = (float)(P.eta2 * P.eta2);
        q.cur1 = (float)(2.0 * P.e1 * P.e1 * c / dx);
        q.cur2 = (float)(2.0 * P.e2 * P.e2 * c / dx);
        q.inv_dx2 = (float)(1.0 / (dx * dx));
        q.inv_dx3 = (float)(1.0 / (dx * dx * dx));
        q.dtau = (float)dt;
        q.dtau_dx = (float)(dt * dx);
        q.aSm1 = (float)(f * (1.0 - delta) / (1.0 + delta) - 1.0);
        q.aGm1 = (float)(f * (1.0 - omega) / (1.0 + omega) - 1.0);
        q.flags = kernel_flags(ctx);
        return U1U1_OK;
    };
    const bool pairs = pairs_enabled(ctx);      // an odd last step takes the one-step kernel
    for (int k = 0; k < n;) {
        const double tk = tau + k * dt;
        StepCoef q, q2;
        double c, delta, omega;
        if (int rc = coef_at(tk, q, c, delta, omega)) return rc;
        if (int rc = prepare_device(ctx)) return rc;      // SM count and tensor maps, once per configure
        int done = 1;
        cudaError_t e;
        if (pairs && k + 1 < n) {
            if (int rc = coef_at(tau + (k + 1) * dt, q2, c, delta, omega)) return rc;
            e = launch_two_steps(ctx, q, q2);
            done = 2;
        } else {
            e = launch_step(ctx, q);
            ctx->cur ^= 1;
        }
        if (e != cudaSuccess) return cuda_fail(ctx, e, "step kernel launch");
        ctx->launches += 1;
        k += done;
        ctx->tau_pos = (tau + (k - 1) * dt) + dt;         // start of the last step taken + dtau
        // weights for the diagnostics of the state just produced
        double a1, c1, d1, o1;
        scalars_at(ctx, ctx->tau_pos, era_m, s, a1, c1, d1, o1);
        ctx->a = a1;
        ctx->c = c1;
        ctx->cG = c * (1.0 + delta) / (1.0 + omega);      // of the last step taken
        invalidate(ctx);
    }
    return U1U1_OK;
}

extern "C" int u1u1_cool(u1u1_ctx *ctx, int32_t n, double dcool)
{
    if (!ctx) return U1U1_EINVAL;
    if (!ctx->configured) return fail(ctx, U1U1_ESTATE, "cool before configure/init_fields");
    if (int rc = cubic_only(ctx, "cool")) return rc;
    if (n < 0 || !(dcool > 0)) return fail(ctx, U1U1_EINVAL, "need n >= 0 and dcool > 0");
    const u1u1_params &P = ctx->prm;
    const double dx = ctx->dx;
    // explicit diffusion: the scalars see 12/dx^2 + lambda sigma^2, the links 12/dx^2 + 2 e^2 sigma^2
    const double lam = std::fmax(std::fmax(P.lambda1 * P.eta1 * P.eta1, P.lambda2 * P.eta2 * P.eta2),
                                 std::fmax(2.0 * P.e1 * P.e1 * P.eta1 * P.eta1, 2.0 * P.e2 * P.e2 * P.eta2 * P.eta2));
    if (dcool * (12.0 / (dx * dx) + lam) >= 2.0)
        return fail(ctx, U1U1_EUNSTABLE, "explicit cooling unstable: need dcool (12/dx^2 + max(lambda, 2 e^2) sigma^2) < 2");
    if (n > 0)
        if (int rc = prepare_device(ctx)) return rc;
    // Pi+ = 0 Pi- + 1 [D-D+ phi - lambda/2 (|phi|^2 - sigma^2) phi], phi += dcool Pi+  (and the same for E, theta)
    StepCoef q;
    q.aS = 0.f; q.bS = 1.f; q.aG = 0.f; q.bG = 1.f; q.aSm1 = -1.f; q.aGm1 = -1.f;
    q.lamh1 = (float)(0.5 * P.lambda1);
    q.lamh2 = (float)(0.5 * P.lambda2);
    q.kap = 0.f;
    q.sig1sq = (float)(P.eta1 * P.eta1);
    q.sig2sq = (float)(P.eta2 * P.eta2);
    q.cur1 = (float)(2.0 * P.e1 * P.e1 / dx);
    q.cur2 = (float)(2.0 * P.e2 * P.e2 / dx);
    q.inv_dx2 = (float)(1.0 / (dx * dx));
    q.inv_dx3 = (float)(1.0 / (dx * dx * dx));
    q.dtau = (float)dcool;
    q.dtau_dx = (float)(dcool * dx);
    q.flags = kernel_flags(ctx);
    const bool pairs = pairs_enabled(ctx);
    for (int k = 0; k < n;) {
        cudaError_t e;
        if (pairs && k + 1 < n) {
            e = launch_two_steps(ctx, q, q);
            k += 2;
        } else {
            e = launch_step(ctx, q);
            ctx->cur ^= 1;
            k += 1;
        }
        if (e != cudaSuccess) return cuda_fail(ctx, e, "cooling kernel launch");
        ctx->launches += 1;
        invalidate(ctx);
    }
    if (n > 0) {
        cudaError_t e = cudaMemsetAsync(mom_buf(ctx), 0, (size_t)NMOM * ctx->V * sizeof(float), ctx->stream);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "cool: zeroing the momenta");
        ctx->a = ctx->c = ctx->cG = 1.0;      // the cooling equations carry no scale factor (Eq. 27-30)
    }
    return U1U1_OK;
}

static DiagCoef diag_coef(const u1u1_ctx *ctx)
{
    const u1u1_params &P = ctx->prm;
    DiagCoef k;
    k.c = ctx->c;
    k.cG = ctx->cG;
    k.inv_dx = 1.0 / ctx->dx;
    k.inv_dx2 = 1.0 / (ctx->dx * ctx->dx);
    k.e1 = P.e1; k.e2 = P.e2; k.lam1 = P.lambda1; k.lam2 = P.lambda2; k.kappa = P.kappa;
    k.sig1sq = P.eta1 * P.eta1; k.sig2sq = P.eta2 * P.eta2;
    return k;
}

static FusedCoef fused_coef(const u1u1_ctx *ctx)
{
    const u1u1_params &P = ctx->prm;
    const double dx = ctx->dx, dx4 = dx * dx * dx * dx;
    FusedCoef k;
    k.inv_dx = 1.0 / dx;
    k.rho1 = 2.0 * P.e1 * P.e1 * ctx->cG;
    k.rho2 = 2.0 * P.e2 * P.e2 * ctx->cG;
    k.inv_dx2 = (float)(1.0 / (dx * dx));
    k.el1 = (float)(1.0 / (2.0 * P.e1 * P.e1));
    k.el2 = (float)(1.0 / (2.0 * P.e2 * P.e2));
    k.mg1 = (float)(1.0 / (2.0 * P.e1 * P.e1 * dx4));
    k.mg2 = (float)(1.0 / (2.0 * P.e2 * P.e2 * dx4));
    k.lam1q = (float)(0.25 * P.lambda1);
    k.lam2q = (float)(0.25 * P.lambda2);
    k.kappa = (float)P.kappa;
    k.sig1sq = (float)(P.eta1 * P.eta1);
    k.sig2sq = (float)(P.eta2 * P.eta2);
    k.c = (float)ctx->c;
    k.inv_c = (float)(1.0 / ctx->c);
    k.flags = kernel_flags(ctx);
    k.nz_own = ctx->nz_own;
    return k;
}

static int fetch(u1u1_ctx *ctx, double *host, int n)
{
    cudaError_t e = cudaMemcpyAsync(host, result(ctx), n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "result readback");
    return U1U1_OK;
}

// per sector: ||g||_2, ||rho||_2, max|g|, ||g||_2 / max(||rho||_2, ||div E||_2, tiny) from [sum g^2, rho^2, div^2] x 2, max|g| x 2
static void gauss_norms(const double *sums, const double *gmax, double *out)
{
    for (int s = 0; s < 2; s++) {
        const double l2g = std::sqrt(sums[3 * s]), l2r = std::sqrt(sums[3 * s + 1]), l2d = std::sqrt(sums[3 * s + 2]);
        out[4 * s + 0] = l2g;
        out[4 * s + 1] = l2r;
        out[4 * s + 2] = gmax[s];
        out[4 * s + 3] = l2g / std::fmax(std::fmax(l2r, l2d), 1e-300);
    }
}

extern "C" int u1u1_gauss_violation(u1u1_ctx *ctx, double *out)
{
    if (!ctx || !out) return ctx ? fail(ctx, U1U1_EINVAL, "out is NULL") : U1U1_EINVAL;
    if (!ctx->configured) return fail(ctx, U1U1_ESTATE, "gauss_violation before configure/init_fields");
    if (int rc = cubic_only(ctx, "gauss_violation")) return rc;
    cudaError_t e = launch_gauss(pos_buf(ctx, ctx->cur), mom_buf(ctx), ctx->V, ctx->N, diag_coef(ctx),
                                 partials(ctx), result(ctx), ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gauss kernel launch");
    ctx->launches += 2;
    double r[8];
    if (int rc = fetch(ctx, r, 8)) return rc;
    gauss_norms(r, r + 6, out);
    return U1U1_OK;
}

// The fused sweep (diag_fused.cu) + the tolerant overlap count; result slots [0, FUSED_NRES) and [32, 34).
// with_codes: also write the winding codes (6 B/site) that u1u1_export_windings decodes.
static int run_sweep(u1u1_ctx *ctx, bool with_codes)
{
    if (int rc = prepare_device(ctx)) return rc;
    DiagMaps maps;
    if (ctx->maps_ready) {
        maps.pos = ctx->pos_halo[ctx->cur];
        maps.mom = ctx->mom_halo[ctx->mcur];
    }
    int nb = 0;
    cudaError_t e = launch_diag_fused(pos_buf(ctx, ctx->cur), mom_buf(ctx), ctx->V, ctx->N, fused_coef(ctx), cells_buf(ctx),
                                      with_codes ? work_buf(ctx) : nullptr, partials(ctx), &nb, ctx->maps_ready ? &maps : nullptr,
                                      ctx->sms, ctx->stream);
    if (e == cudaSuccess) e = launch_fold(partials(ctx), nb, FUSED_NRES, FUSED_NSUM, result(ctx), ctx->stream);
    if (e == cudaSuccess) e = launch_overlap_tol(cells_buf(ctx), ctx->V, ctx->N, partials(ctx), result(ctx) + 32, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "diagnostics kernel launch");
    ctx->launches += 4;
    ctx->diag_valid = true;
    ctx->codes_valid = with_codes;
    ctx->labels_valid = false;
    return U1U1_OK;
}

// out slots from the raw sums r[0 .. FUSED_NRES) of the sweep and the tolerant counts r[32], r[33] over `sites` sites
static void derive_diagnostics(const u1u1_ctx *ctx, const double *r, double sites, double *out)
{
    memset(out, 0, U1U1_DIAG_LEN * sizeof(double));
    const double dx = ctx->dx, vol = sites * dx * dx * dx;
    out[U1U1_D_TAU] = ctx->tau_pos;
    out[U1U1_D_A] = ctx->a;
    out[U1U1_D_C] = ctx->c;
    out[U1U1_D_SUMW_P] = r[FR_SUMW];
    out[U1U1_D_SUMW_Q] = r[FR_SUMW + 1];
    out[U1U1_D_NEAR_P] = r[FR_NEAR];
    out[U1U1_D_NEAR_Q] = r[FR_NEAR + 1];
    out[U1U1_D_MAXW] = r[FR_MAXW];
    out[U1U1_D_CELLS_P] = r[FR_CELLS];
    out[U1U1_D_CELLS_Q] = r[FR_CELLS + 1];
    out[U1U1_D_CELLS_PQ] = r[FR_CELLS + 2];
    const double *dn = r + FR_DENS;      // sum L, kin L, grad L, kin V, grad V, V, kin, grad, elec, mag, pot
    for (int k = 0; k < 11; k++) out[U1U1_D_SUM_L + k] = dn[k];
    // derived scalars, Eq. 31-37; L_pq = dx N_pq, L_p = dx sum|W^p| - L_pq (:188)
    const double L_pq = dx * r[FR_CELLS + 2], L_p = dx * r[FR_SUMW] - L_pq, L_q = dx * r[FR_SUMW + 1] - L_pq, tot = L_pq + L_p + L_q;
    const double inf = INFINITY;
    out[U1U1_D_L_P] = L_p;
    out[U1U1_D_L_Q] = L_q;
    out[U1U1_D_L_PQ] = L_pq;
    out[U1U1_D_XI_P] = L_p > 0 ? std::sqrt(vol / L_p) : inf;
    out[U1U1_D_XI_Q] = L_q > 0 ? std::sqrt(vol / L_q) : inf;
    out[U1U1_D_XI_PQ] = L_pq > 0 ? std::sqrt(vol / L_pq) : inf;
    out[U1U1_D_XI_W] = tot > 0 ? std::sqrt(vol / tot) : inf;
    const double mu = 2.0 * 3.14159265358979323846 * ctx->prm.eta1 * ctx->prm.eta1;
    const double sumL = dx * dx * dx * dn[0];
    out[U1U1_D_XI_L] = sumL < 0 ? std::sqrt(-mu * vol / sumL) : NAN;
    out[U1U1_D_F_TOTAL] = tot > 0 ? L_pq / tot : 0.0;
    out[U1U1_D_F_P] = L_p > 0 ? L_pq / L_p : 0.0;
    const double RL = dn[2] != 0 ? dn[1] / dn[2] : NAN, RV = dn[4] != 0 ? dn[3] / dn[4] : NAN;
    out[U1U1_D_V2_L] = 2.0 * RL / (1.0 + RL);
    out[U1U1_D_V2_PQ] = 2.0 * RV / (1.0 + RV);
    // a velocity only while the weight localises on strings: R finite, 0 <= R <= 1 (NaN fails both comparisons)
    out[U1U1_D_V2_VALID] = (RL >= 0.0 && RL <= 1.0 ? 1.0 : 0.0) + (RV >= 0.0 && RV <= 1.0 ? 2.0 : 0.0);
    out[U1U1_D_ENERGY] = dx * dx * dx * (dn[6] + dn[7] + dn[8] + dn[9] + dn[10]);
    out[U1U1_D_CELLS_PQ_TOL_P] = r[32];
    out[U1U1_D_CELLS_PQ_TOL_Q] = r[33];
    out[U1U1_D_L_PQ_TOL] = 0.5 * dx * (r[32] + r[33]);
    out[U1U1_D_MAX_THETA] = r[FR_MAXTH];
    gauss_norms(r + FR_GAUSS, r + FR_GMAX, out + U1U1_D_GAUSS);
}

extern "C" int u1u1_diagnostics(u1u1_ctx *ctx, double *out)
{
    if (!ctx || !out) return ctx ? fail(ctx, U1U1_EINVAL, "out is NULL") : U1U1_EINVAL;
    if (!ctx->configured) return fail(ctx, U1U1_ESTATE, "diagnostics before configure/init_fields");
    if (int rc = cubic_only(ctx, "diagnostics")) return rc;
    if (int rc = run_sweep(ctx, false)) return rc;
    double r[34];
    if (int rc = fetch(ctx, r, 34)) return rc;
    // the byte lanes of the winding sweep hold wrap counts |n| <= 31: fail loudly beyond (non-compact links, reading R-9)
    ctx->last_max_theta = std::fmax(ctx->last_max_theta, r[FR_MAXTH]);
    if (r[FR_MAXTH] > 180.0) {
        ctx->diag_valid = false;
        return fail(ctx, U1U1_ESTATE, "diagnostics: a link phase exceeds |theta| = 180, beyond the range of the winding sweep");
    }
    derive_diagnostics(ctx, r, (double)ctx->V, out);
    return U1U1_OK;
}

static int relayout(u1u1_ctx *ctx, float *canon, int to_canonical)
{
    cudaError_t e = launch_relayout(pos_buf(ctx, ctx->cur), mom_buf(ctx), canon, ctx->V, ctx->V, 0, 0, 20, to_canonical, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "relayout kernel launch");
    ctx->launches += 1;
    if (!to_canonical) invalidate(ctx);
    return U1U1_OK;
}

extern "C" int u1u1_export_state(u1u1_ctx *ctx, void *dst_dev)
{
    if (!ctx || !dst_dev) return ctx ? fail(ctx, U1U1_EINVAL, "dst is NULL") : U1U1_EINVAL;
    if (!ctx->configured) return fail(ctx, U1U1_ESTATE, "export_state before configure/init_fields");
    if (int rc = cubic_only(ctx, "export_state")) return rc;
    return relayout(ctx, (float *)dst_dev, 1);
}

extern "C" int u1u1_import_state(u1u1_ctx *ctx, const void *src_dev)
{
    if (!ctx || !src_dev) return ctx ? fail(ctx, U1U1_EINVAL, "src is NULL") : U1U1_EINVAL;
    if (!ctx->configured) return fail(ctx, U1U1_ESTATE, "import_state before configure");
    if (int rc = cubic_only(ctx, "import_state")) return rc;
    return relayout(ctx, (float *)src_dev, 0);
}

extern "C" int u1u1_import_state_tiled(u1u1_ctx *ctx, const void *src_dev, int32_t n_src)
{
    if (!ctx || !src_dev) return ctx ? fail(ctx, U1U1_EINVAL, "src is NULL") : U1U1_EINVAL;
    if (!ctx->configured) return fail(ctx, U1U1_ESTATE, "import_state_tiled before configure");
    if (int rc = cubic_only(ctx, "import_state_tiled")) return rc;
    if (n_src < 1 || ctx->N % n_src != 0) return fail(ctx, U1U1_ESIZE, "N must be a multiple of n_src");
    cudaError_t e = launch_import_tiled(pos_buf(ctx, ctx->cur), mom_buf(ctx), (const float *)src_dev, ctx->V, ctx->N, n_src, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "import_state_tiled launch");
    ctx->launches += 1;
    invalidate(ctx);
    return U1U1_OK;
}

extern "C" int u1u1_export_block(u1u1_ctx *ctx, int32_t x0, int32_t y0, int32_t z0, int32_t bx, int32_t by,
                                 int32_t bz, void *dst_dev)
{
    if (!ctx || !dst_dev) return ctx ? fail(ctx, U1U1_EINVAL, "dst is NULL") : U1U1_EINVAL;
    if (!ctx->configured) return fail(ctx, U1U1_ESTATE, "export_block before configure/init_fields");
    if (int rc = cubic_only(ctx, "export_block")) return rc;
    if (bx < 1 || by < 1 || bz < 1 || bx > ctx->N || by > ctx->N || bz > ctx->N)
        return fail(ctx, U1U1_EINVAL, "block extents must lie in [1, N]");
    cudaError_t e = launch_export_block(pos_buf(ctx, ctx->cur), mom_buf(ctx), ctx->V, ctx->N, x0, y0, z0, bx, by,
                                        bz, (float *)dst_dev, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "export_block launch");
    ctx->launches += 1;
    return U1U1_OK;
}

// Host variants: one canonical component at a time is gathered into (scattered from) one of two staging planes in
// the scratch work area by the relayout kernel, and moved by cudaMemcpyAsync on a second stream, so that the kernel
// of component c+1 overlaps the PCIe copy of component c and no second full-size device buffer is needed (a canonical
// copy of a 1024^3 state would not fit beside the state).  Clobbers the winding codes / segment labels, not the cells.
static int host_copy(u1u1_ctx *ctx, void *host, int to_host)
{
    const size_t V = ctx->V, bytes = V * sizeof(float);
    cudaError_t e = cudaSuccess;
    if (!ctx->copy_stream) {
        e = cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking);
        for (int b = 0; b < 2 && e == cudaSuccess; b++) {
            e = cudaEventCreateWithFlags(&ctx->ev_kernel[b], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_copy[b], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) return cuda_fail(ctx, e, "host copy: creating the copy stream");
    }
    ctx->codes_valid = ctx->labels_valid = false;
    if (!to_host) ctx->diag_valid = false;
    float *stage[2] = {(float *)work_buf(ctx), (float *)work_buf(ctx) + V};
    cudaStream_t ms = ctx->stream, cs = ctx->copy_stream;
    // the copy stream starts after everything already queued on the caller's stream
    e = cudaEventRecord(ctx->ev_kernel[0], ms);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(cs, ctx->ev_kernel[0], 0);
    for (int c = 0; c < 20 && e == cudaSuccess; c++) {
        const int b = c & 1;
        float *h = (float *)host + (size_t)c * V;
        if (to_host) {
            if (c >= 2) e = cudaStreamWaitEvent(ms, ctx->ev_copy[b], 0);              // staging plane b is free again
            if (e == cudaSuccess) e = launch_relayout(pos_buf(ctx, ctx->cur), mom_buf(ctx), stage[b], V, V, 0, c, 1, 1, ms);
            if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_kernel[b], ms);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(cs, ctx->ev_kernel[b], 0);
            if (e == cudaSuccess) e = cudaMemcpyAsync(h, stage[b], bytes, cudaMemcpyDeviceToHost, cs);
            if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_copy[b], cs);
        } else {
            if (c >= 2) e = cudaStreamWaitEvent(cs, ctx->ev_kernel[b], 0);            // its scatter kernel has run
            if (e == cudaSuccess) e = cudaMemcpyAsync(stage[b], h, bytes, cudaMemcpyHostToDevice, cs);
            if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_copy[b], cs);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(ms, ctx->ev_copy[b], 0);
            if (e == cudaSuccess) e = launch_relayout(pos_buf(ctx, ctx->cur), mom_buf(ctx), stage[b], V, V, 0, c, 1, 0, ms);
            if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_kernel[b], ms);
        }
        ctx->launches += 1;
    }
    for (int b = 0; b < 2 && e == cudaSuccess; b++) e = cudaStreamWaitEvent(ms, ctx->ev_copy[b], 0);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ms);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "host<->device state copy");
    return U1U1_OK;
}

extern "C" int u1u1_export_state_host(u1u1_ctx *ctx, void *dst_host)
{
    if (!ctx || !dst_host) return ctx ? fail(ctx, U1U1_EINVAL, "dst is NULL") : U1U1_EINVAL;
    if (!ctx->configured) return fail(ctx, U1U1_ESTATE, "export_state_host before configure/init_fields");
    if (int rc = cubic_only(ctx, "export_state_host")) return rc;
    return host_copy(ctx, dst_host, 1);
}

extern "C" int u1u1_import_state_host(u1u1_ctx *ctx, const void *src_host)
{
    if (!ctx || !src_host) return ctx ? fail(ctx, U1U1_EINVAL, "src is NULL") : U1U1_EINVAL;
    if (!ctx->configured) return fail(ctx, U1U1_ESTATE, "import_state_host before configure");
    if (int rc = cubic_only(ctx, "import_state_host")) return rc;
    return host_copy(ctx, const_cast<void *>(src_host), 0);
}

extern "C" int u1u1_pq_segments(u1u1_ctx *ctx, int32_t min_cells, int32_t tolerant, double *out)
{
    if (!ctx || !out) return ctx ? fail(ctx, U1U1_EINVAL, "out is NULL") : U1U1_EINVAL;
    if (min_cells < 1 || (tolerant != 0 && tolerant != 1)) return fail(ctx, U1U1_EINVAL, "need min_cells >= 1 and tolerant in {0, 1}");
    if (!ctx->diag_valid) return fail(ctx, U1U1_ESTATE, "pq_segments needs u1u1_diagnostics on the current state first");
    const size_t V = ctx->V;
    // scratch work area: [labels 4V | sizes 4V]; the cell arrays in front of it are only read
    int *label = (int *)work_buf(ctx), *size = (int *)(work_buf(ctx) + 4 * V);
    cudaError_t e = launch_segments(cells_buf(ctx), V, ctx->N, tolerant, min_cells, label, size, partials(ctx), result(ctx),
                                    ctx->stream);
    ctx->codes_valid = false;
    ctx->labels_valid = false;
    if (e != cudaSuccess) return cuda_fail(ctx, e, "pq_segments kernel launch");
    ctx->launches += 5;
    double r[7];
    if (int rc = fetch(ctx, r, 7)) return rc;
    ctx->labels_valid = true;
    memset(out, 0, U1U1_SEG_LEN * sizeof(double));
    out[0] = r[0];
    out[1] = ctx->dx * r[1];
    out[2] = r[0] > 0 ? out[1] / r[0] : 0.0;
    out[3] = r[2];
    out[4] = r[3];
    out[5] = r[4];
    out[6] = r[6];
    out[7] = r[5];
    return U1U1_OK;
}

extern "C" int u1u1_export_labels(u1u1_ctx *ctx, void *labels_dev)
{
    if (!ctx || !labels_dev) return ctx ? fail(ctx, U1U1_EINVAL, "dst is NULL") : U1U1_EINVAL;
    if (!ctx->labels_valid) return fail(ctx, U1U1_ESTATE, "export_labels needs u1u1_pq_segments on the current state first");
    cudaError_t e = cudaMemcpyAsync(labels_dev, work_buf(ctx), ctx->V * sizeof(int), cudaMemcpyDeviceToDevice, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "labels copy");
    return U1U1_OK;
}

extern "C" int u1u1_export_windings(u1u1_ctx *ctx, int32_t sector, void *w_dev, void *near_dev, void *cells_dev)
{
    if (!ctx) return U1U1_EINVAL;
    if (sector != 0 && sector != 1) return fail(ctx, U1U1_EINVAL, "sector must be 0 or 1");
    if (!ctx->diag_valid) return fail(ctx, U1U1_ESTATE, "export_windings needs u1u1_diagnostics on the current state first");
    const size_t V = ctx->V;
    if (w_dev || near_dev) {
        // the sweep writes the per-plaquette codes (6 B/site) only on request: run it again in export mode
        if (!ctx->codes_valid)
            if (int rc = run_sweep(ctx, true)) return rc;
        cudaError_t e = launch_decode_windings(work_buf(ctx) + (size_t)3 * sector * V, 3 * V, (int8_t *)w_dev,
                                               (uint8_t *)near_dev, ctx->stream);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "decode_windings launch");
        ctx->launches += 1;
    }
    if (cells_dev) {
        cudaError_t e = cudaMemcpyAsync(cells_dev, cells_buf(ctx) + (size_t)sector * V, V, cudaMemcpyDeviceToDevice, ctx->stream);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "cells copy");
    }
    return U1U1_OK;
}

// ---- z slabs: one lattice split over several GPUs (SURVEY.md 8(f)-4 "then z-slab multi-GPU") -------
static bool slab_ok(int32_t N, int32_t nz_own) { return N >= 8 && N <= 8192 && (N % 4) == 0 && nz_own >= 1 && nz_own <= 8192; }

extern "C" size_t u1u1_slab_state_bytes(int32_t N, int32_t nz_own)
{
    if (!slab_ok(N, nz_own)) return 0;
    return (size_t)(2 * NPOS + NMOM) * (size_t)N * N * (size_t)(nz_own + 2) * sizeof(float);
}

extern "C" int u1u1_configure_slab(u1u1_ctx *ctx, int32_t N, int32_t nz_own, int64_t z_first, double dx, const u1u1_params *params)
{
    if (!ctx) return U1U1_EINVAL;
    if (!slab_ok(N, nz_own) || z_first < 0) return fail(ctx, U1U1_ESIZE, "slab: N a multiple of 4 in [8, 8192], 1 <= nz_own <= 8192, z_first >= 0");
    if (!(dx > 0)) return fail(ctx, U1U1_EINVAL, "dx must be positive");
    if (int rc = check_params(ctx, params)) return rc;
    if (ctx->state_bytes < u1u1_slab_state_bytes(N, nz_own)) return fail(ctx, U1U1_ESIZE, "state buffer smaller than u1u1_slab_state_bytes(N, nz_own)");
    ctx->N = N;
    ctx->V = (size_t)N * N * (size_t)(nz_own + 2);
    ctx->nz_own = nz_own;
    ctx->z_first = z_first;
    ctx->peer_up = ctx->peer_dn = nullptr;
    ctx->dx = dx;
    ctx->prm = *params;
    ctx->configured = true;
    ctx->cur = 0;
    ctx->mcur = 0;
    ctx->tau_pos = params->tau_norm;
    ctx->a = ctx->c = ctx->cG = 1.0;
    invalidate(ctx);
    ctx->maps_ready = false;
    return U1U1_OK;
}

extern "C" int u1u1_set_slab_peers(u1u1_ctx *ctx, void *up_state_dev, void *dn_state_dev)
{
    if (!ctx) return U1U1_EINVAL;
    if (!ctx->nz_own) return fail(ctx, U1U1_ESTATE, "set_slab_peers needs u1u1_configure_slab first");
    if (!up_state_dev || !dn_state_dev) return fail(ctx, U1U1_EINVAL, "peer state buffers must not be NULL");
    ctx->peer_up = (float *)up_state_dev;
    ctx->peer_dn = (float *)dn_state_dev;
    return U1U1_OK;
}

extern "C" int u1u1_init_slab(u1u1_ctx *ctx, uint64_t seed)
{
    if (!ctx) return U1U1_EINVAL;
    if (!ctx->nz_own) return fail(ctx, U1U1_ESTATE, "init_slab needs u1u1_configure_slab first");
    if (ctx->prm.init_kind != 0) return fail(ctx, U1U1_EINVAL, "init_slab generates the random-phase initial condition only (init_kind 0)");
    const size_t NN = (size_t)ctx->N * ctx->N;
    cudaError_t e = cudaMemsetAsync(ctx->state, 0, u1u1_slab_state_bytes(ctx->N, ctx->nz_own), ctx->stream);
    if (e == cudaSuccess)
        e = launch_init_random_phase(pos_buf(ctx, 0), NN * ctx->nz_own, NN, NN * (size_t)ctx->z_first, seed, ctx->prm.eta1,
                                     ctx->prm.eta2, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "init_slab");
    ctx->launches += 1;
    ctx->cur = 0;
    return U1U1_OK;
}

static int slab_relayout(u1u1_ctx *ctx, float *canon, int to_canonical)
{
    const size_t NN = (size_t)ctx->N * ctx->N;
    cudaError_t e = launch_relayout(pos_buf(ctx, ctx->cur), mom_buf(ctx), canon, ctx->V, NN * ctx->nz_own, NN, 0, 20, to_canonical,
                                    ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "slab relayout launch");
    ctx->launches += 1;
    return U1U1_OK;
}

extern "C" int u1u1_export_slab(u1u1_ctx *ctx, void *dst_dev)
{
    if (!ctx || !dst_dev) return ctx ? fail(ctx, U1U1_EINVAL, "dst is NULL") : U1U1_EINVAL;
    if (!ctx->nz_own) return fail(ctx, U1U1_ESTATE, "export_slab needs u1u1_configure_slab first");
    return slab_relayout(ctx, (float *)dst_dev, 1);
}

extern "C" int u1u1_import_slab(u1u1_ctx *ctx, const void *src_dev)
{
    if (!ctx || !src_dev) return ctx ? fail(ctx, U1U1_EINVAL, "src is NULL") : U1U1_EINVAL;
    if (!ctx->nz_own) return fail(ctx, U1U1_ESTATE, "import_slab needs u1u1_configure_slab first");
    return slab_relayout(ctx, (float *)src_dev, 0);
}

// my boundary planes of the CURRENT positions -> the neighbours' halo planes (needed once, after init / import: from
// then on every step writes them itself).  Three contiguous chunks per plane (packs A, B, C).
extern "C" int u1u1_push_halos(u1u1_ctx *ctx)
{
    if (!ctx) return U1U1_EINVAL;
    if (!ctx->nz_own || !ctx->peer_up || !ctx->peer_dn) return fail(ctx, U1U1_ESTATE, "push_halos needs u1u1_configure_slab and u1u1_set_slab_peers first");
    const size_t NN = (size_t)ctx->N * ctx->N, V = ctx->V, off = (size_t)ctx->cur * NPOS * V;
    const float *mine = pos_buf(ctx, ctx->cur);
    float *up = ctx->peer_up + off, *dn = ctx->peer_dn + off;
    const size_t top = (size_t)ctx->nz_own, bot = 1, up_halo = 0, dn_halo = (size_t)ctx->nz_own + 1;
    cudaError_t e = cudaSuccess;
    for (int pack = 0; pack < 3 && e == cudaSuccess; pack++) {
        const size_t base = pack == 0 ? 0 : pack == 1 ? 4 * V : 8 * V, w = pack == 2 ? 2 : 4;     // floats per site
        e = cudaMemcpyAsync(up + base + w * NN * up_halo, mine + base + w * NN * top, w * NN * sizeof(float), cudaMemcpyDeviceToDevice, ctx->stream);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(dn + base + w * NN * dn_halo, mine + base + w * NN * bot, w * NN * sizeof(float), cudaMemcpyDeviceToDevice, ctx->stream);
    }
    if (e != cudaSuccess) return cuda_fail(ctx, e, "push_halos");
    return U1U1_OK;
}

// Diagnostics of a lattice in z slabs: every rank sweeps its own planes (u1u1_slab_diagnostics_partial), the ranks add the
// first U1U1_SLAB_NSUM raw values and take the maximum of the rest, and any rank turns the reduced array into the
// u1u1_diagnostics output (u1u1_slab_diagnostics_finish).  Before the sweep the momentum pack C of the plane below must
// be in place (u1u1_push_diag_halos on every rank, then a barrier); the positions' upper halo is there from the step.
extern "C" int u1u1_push_diag_halos(u1u1_ctx *ctx)
{
    if (!ctx) return U1U1_EINVAL;
    if (!ctx->nz_own || !ctx->peer_up || !ctx->peer_dn) return fail(ctx, U1U1_ESTATE, "push_diag_halos needs u1u1_configure_slab and u1u1_set_slab_peers first");
    const size_t NN = (size_t)ctx->N * ctx->N, V = ctx->V, moff = (size_t)2 * NPOS * V + 8 * V;       // pack C of the momenta
    // my top own plane of (E_z, H_z) -> plane 0 of the slab above
    cudaError_t e = cudaMemcpyAsync(ctx->peer_up + moff, ctx->state + moff + 2 * NN * (size_t)ctx->nz_own, 2 * NN * sizeof(float),
                                    cudaMemcpyDeviceToDevice, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "push_diag_halos");
    return U1U1_OK;
}

extern "C" size_t u1u1_slab_scratch_bytes(int32_t N, int32_t nz_own)
{
    if (!slab_ok(N, nz_own)) return 0;
    const size_t Vb = (size_t)N * N * (size_t)(nz_own + 2);
    return ((2 * Vb + 255) / 256) * 256 + ((size_t)RED_MAX_BLOCKS * RED_SLOTS + 64) * sizeof(double);
}

extern "C" int u1u1_slab_diagnostics_partial(u1u1_ctx *ctx, double *raw)
{
    if (!ctx || !raw) return ctx ? fail(ctx, U1U1_EINVAL, "raw is NULL") : U1U1_EINVAL;
    if (!ctx->nz_own) return fail(ctx, U1U1_ESTATE, "slab_diagnostics_partial needs u1u1_configure_slab first");
    if (ctx->scratch_bytes < u1u1_slab_scratch_bytes(ctx->N, ctx->nz_own)) return fail(ctx, U1U1_ESIZE, "scratch buffer smaller than u1u1_slab_scratch_bytes(N, nz_own)");
    if (int rc = prepare_device(ctx)) return rc;
    // slab scratch: [cells 2 V_buf] pad-> [partials][result]
    double *part = (double *)(ctx->scratch + ((2 * ctx->V + 255) / 256) * 256), *res = part + (size_t)RED_MAX_BLOCKS * RED_SLOTS;
    DiagMaps maps;
    if (ctx->maps_ready) {
        maps.pos = ctx->pos_halo[ctx->cur];
        maps.mom = ctx->mom_halo[ctx->mcur];
    }
    int nb = 0;
    cudaError_t e = launch_diag_fused(pos_buf(ctx, ctx->cur), mom_buf(ctx), ctx->V, ctx->N, fused_coef(ctx), ctx->scratch, nullptr, part,
                                      &nb, ctx->maps_ready ? &maps : nullptr, ctx->sms, ctx->stream);
    if (e == cudaSuccess) e = launch_fold(part, nb, FUSED_NRES, FUSED_NSUM, res, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "slab diagnostics kernel launch");
    ctx->launches += 2;
    e = cudaMemcpyAsync(raw, res, FUSED_NRES * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "slab diagnostics readback");
    return U1U1_OK;
}

extern "C" int u1u1_slab_diagnostics_finish(u1u1_ctx *ctx, const double *raw_reduced, int64_t nz_global, double *out)
{
    if (!ctx || !raw_reduced || !out) return ctx ? fail(ctx, U1U1_EINVAL, "NULL argument") : U1U1_EINVAL;
    if (!ctx->nz_own || nz_global < ctx->nz_own) return fail(ctx, U1U1_ESTATE, "slab_diagnostics_finish needs a slab context and the global number of planes");
    if (raw_reduced[FR_MAXTH] > 180.0)
        return fail(ctx, U1U1_ESTATE, "diagnostics: a link phase exceeds |theta| = 180, beyond the range of the winding sweep");
    double r[34];
    for (int k = 0; k < FUSED_NRES; k++) r[k] = raw_reduced[k];
    for (int k = FUSED_NRES; k < 34; k++) r[k] = NAN;        // the tolerant overlap needs cell-array halos: not on slabs
    derive_diagnostics(ctx, r, (double)ctx->N * ctx->N * (double)nz_global, out);
    return U1U1_OK;
}

// api.cu -- the C ABI of libwoden_b200.so (include/woden_b200.h): argument validation, the
// context's grow-only device scratch, the per-call channel table, and kernel sequencing.
// Host code only; every step of the hot path runs in the kernels it launches.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include <cuda_fp16.h>

#include "../../include/woden_b200.h"
#include "kernels.h"

using namespace woden;

unsigned long long woden::g_kernel_launches = 0;

namespace {

struct DevBuf {
    void *p = nullptr;
    size_t cap = 0;
    cudaError_t reserve(size_t bytes)
    {
        if (bytes <= cap) return cudaSuccess;
        if (p) { cudaFree(p); p = nullptr; cap = 0; }
        size_t want = bytes + bytes / 8 + 256;
        cudaError_t e = cudaMalloc(&p, want);
        if (e == cudaSuccess) cap = want;
        return e;
    }
    void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
};

}  // namespace

struct woden_ctx {
    int device = 0;
    int path = WODEN_PATH_AUTO;
    int last_path = WODEN_PATH_NONE;
    cudaStream_t last_stream = nullptr;
    std::string last_error;
    DevBuf geo, flux, tri, chan, err, hang, bmat, bscale, lut, wblocks;
    DevBuf f_hx, f_a0, f_at, f_small, f_gram, f_ops, f_part;     // woden_fit_shapelets scratch
    DevBuf t_list, t_sums;                                       // woden_shapelet_truncation_weights staging
    int lut_pm = -1, lut_nx = 0;
    double lut_dx = 0.0;
    int shapelet_path = WODEN_SHAPELET_AUTO;
    int last_shapelet_path = WODEN_PATH_NONE, last_shapelet_bucket = -1;
    std::vector<double> chan_freqs;      // frequencies the device channel table was built from
    std::vector<double> chan_s_host;     // nu_f / c of the padded channel list (host copy)
    cudaStream_t walk_stream = nullptr;  // second lane of the channel-walking launches
    cudaEvent_t walk_fork = nullptr, walk_join = nullptr;
    void (*walk_tile_done)(void *, int, cudaStream_t) = nullptr;   // set by woden_simulate_host around its last call
    void *walk_tile_user = nullptr;
    std::vector<cudaEvent_t> tile_events;
    cudaEvent_t fit_t0 = nullptr, fit_t1 = nullptr;   // around the last fit's Gram kernel
    int chan_F_pad = 0;
    ChanTable ch{};
    // woden_simulate_host staging
    DevBuf h_uvw, h_comp, h_int, h_vis;
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t chunk_done[8] = {};
};

namespace {

constexpr int SHAPELET_TENSOR_MIN_ORDER = 24;   // order bucket from which the tensor path measured faster (profiles/shapelet_mma_r2.md)
constexpr int SIM_CHUNKS = 8;   // time chunks of woden_simulate_host (compute / copy-back overlap)
constexpr int CHAN_TILE = 32;   // F_pad granularity: lcm of the kernels' channel tiles
constexpr int WALK_MIN_F = 8;   // shorter channel lists take the general path

int fail_cuda(woden_ctx *ctx, cudaError_t e, const char *where)
{
    ctx->last_error = std::string(where) + ": " + cudaGetErrorString(e);
    cudaGetLastError();
    return WODEN_ERR_CUDA;
}

#define CU(ctx, call, where)                                                     \
    do {                                                                         \
        cudaError_t e__ = (call);                                                \
        if (e__ != cudaSuccess) return fail_cuda((ctx), e__, (where));           \
    } while (0)

int check_uvw(const woden_uvw *uvw)
{
    if (!uvw || !uvw->u_m || !uvw->v_m || !uvw->w_m || !uvw->freqs_hz) return WODEN_ERR_NULL;
    if (uvw->n_baselines <= 0 || uvw->n_times <= 0 || uvw->n_freqs <= 0) return WODEN_ERR_DIM;
    if (uvw->n_freqs > 65535 * 1) return WODEN_ERR_DIM;                  // grid.y of the shapelet kernel
    for (int f = 0; f < uvw->n_freqs; ++f)
        if (!(uvw->freqs_hz[f] > 0.0) || !std::isfinite(uvw->freqs_hz[f])) return WODEN_ERR_DIM;
    return WODEN_OK;
}

int ensure_err(woden_ctx *ctx, cudaStream_t st)
{
    if (!ctx->err.p) {
        CU(ctx, ctx->err.reserve(sizeof(unsigned int)), "alloc error counter");
        CU(ctx, cudaMemsetAsync(ctx->err.p, 0, sizeof(unsigned int), st), "clear error counter");
    }
    return WODEN_OK;
}

// Build (or reuse) the device channel table for this frequency list (step S1 constants).
int ensure_chan(woden_ctx *ctx, const woden_uvw *uvw, cudaStream_t st)
{
    const int F = uvw->n_freqs;
    if ((int)ctx->chan_freqs.size() == F && ctx->chan.p &&
        std::memcmp(ctx->chan_freqs.data(), uvw->freqs_hz, sizeof(double) * F) == 0)
        return WODEN_OK;
    const int F_pad = (F + CHAN_TILE - 1) / CHAN_TILE * CHAN_TILE;
    const size_t bytes = (size_t)F_pad * (8 + 8 + 4);
    std::vector<unsigned char> host(bytes, 0);
    double *s = reinterpret_cast<double *>(host.data());
    double *nu = s + F_pad;
    float *ns2 = reinterpret_cast<float *>(nu + F_pad);
    for (int f = 0; f < F; ++f) {
        nu[f] = uvw->freqs_hz[f];
        s[f] = nu[f] / C_LIGHT;
        ns2[f] = (float)(-(s[f] * s[f]));
    }
    // Channel-walking eligibility: an arithmetic progression (to 1e-9 of the step) of at least
    // WALK_MIN_F channels whose continuation over the padded tiles stays positive and whose chains
    // (seed +- 8 steps) span at most +-12.5 % in frequency.  The last condition is what keeps the
    // Gaussian envelope walk exact where its seed has flushed to zero (predict_walk.cu) and keeps
    // short, widely spaced lists (which would mostly fill the 32-channel tiles with padding) on the
    // general path.
    int uniform = 0;
    double ds = 0.0;
    if (F >= WALK_MIN_F) {
        const double d = uvw->freqs_hz[1] - uvw->freqs_hz[0];
        uniform = d != 0.0;
        for (int f = 0; f < F && uniform; ++f)
            if (std::fabs(uvw->freqs_hz[f] - (uvw->freqs_hz[0] + f * d)) > 1e-9 * std::fabs(d)) uniform = 0;
        const double nu_lo = std::fmin(uvw->freqs_hz[0], uvw->freqs_hz[0] + (F_pad - 1) * d);
        if (!(nu_lo > 0.0) || (WALK_FT / 4) * std::fabs(d) > 0.125 * nu_lo) uniform = 0;
        ds = d / C_LIGHT;
    }
    // the channel-walking kernel seeds its chains at fixed tile positions, which may lie past F in
    // the last tile: continue the (uniform) grid there; those channels are computed, never stored
    if (uniform)
        for (int f = F; f < F_pad; ++f) s[f] = (uvw->freqs_hz[0] + f * (uvw->freqs_hz[1] - uvw->freqs_hz[0])) / C_LIGHT;
    ctx->chan_freqs.clear();
    CU(ctx, ctx->chan.reserve(bytes), "alloc channel table");
    // pageable source: the runtime stages it before returning, so `host` may die afterwards
    CU(ctx, cudaMemcpyAsync(ctx->chan.p, host.data(), bytes, cudaMemcpyHostToDevice, st), "upload channel table");
    ctx->chan_freqs.assign(uvw->freqs_hz, uvw->freqs_hz + F);
    ctx->chan_F_pad = F_pad;
    ctx->chan_s_host.assign(s, s + F_pad);
    ctx->ch.s_host = ctx->chan_s_host.data();
    ctx->ch.s = reinterpret_cast<const double *>(ctx->chan.p);
    ctx->ch.nu = ctx->ch.s + F_pad;
    ctx->ch.ns2 = reinterpret_cast<const float *>(ctx->ch.nu + F_pad);
    ctx->ch.F = F;
    ctx->ch.F_pad = F_pad;
    ctx->ch.uniform = uniform;
    ctx->ch.ds = ds;
    return WODEN_OK;
}

int ensure_walk_streams(woden_ctx *ctx)
{
    if (ctx->walk_stream) return WODEN_OK;
    CU(ctx, cudaStreamCreateWithFlags(&ctx->walk_stream, cudaStreamNonBlocking), "create walk stream");
    CU(ctx, cudaEventCreateWithFlags(&ctx->walk_fork, cudaEventDisableTiming), "create event");
    CU(ctx, cudaEventCreateWithFlags(&ctx->walk_join, cudaEventDisableTiming), "create event");
    return WODEN_OK;
}

int zero_or_nothing(woden_ctx *ctx, const woden_uvw *uvw, float *vis, int accumulate, cudaStream_t st)
{
    if (!accumulate) {
        const size_t bytes = (size_t)uvw->n_times * uvw->n_freqs * uvw->n_baselines * 8;
        CU(ctx, cudaMemsetAsync(vis, 0, bytes, st), "zero-fill vis");
    }
    return WODEN_OK;
}

struct Bind {
    woden_ctx *ctx;
    int prev = -1;
    bool ok = true;
    explicit Bind(woden_ctx *c) : ctx(c)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; cudaGetLastError(); return; }
        if (prev != c->device && cudaSetDevice(c->device) != cudaSuccess) { ok = false; cudaGetLastError(); }
    }
    ~Bind() { if (ok && prev >= 0 && prev != ctx->device) cudaSetDevice(prev); }
};

int common_checks(woden_ctx *ctx, const woden_uvw *uvw, int n, const double *l, const double *m,
                  const double *s0, const double *alpha, double ref_freq, const float *vis)
{
    if (!ctx) return WODEN_ERR_NULL;
    int rc = check_uvw(uvw);
    if (rc != WODEN_OK) return rc;
    if (!vis) return WODEN_ERR_NULL;
    if (n < 0) return WODEN_ERR_DIM;
    if (n > 0 && (!l || !m || !s0 || !alpha)) return WODEN_ERR_NULL;
    if (!(ref_freq > 0.0) || !std::isfinite(ref_freq)) return WODEN_ERR_DIM;
    if ((long long)uvw->n_times * uvw->n_baselines > (1LL << 38)) return WODEN_ERR_DIM;
    return WODEN_OK;
}

}  // namespace

extern "C" {

int woden_create(woden_ctx **out, int cuda_device)
{
    if (!out) return WODEN_ERR_NULL;
    *out = nullptr;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || cuda_device < 0 || cuda_device >= count) {
        cudaGetLastError();
        return WODEN_ERR_CUDA;
    }
    woden_ctx *ctx = new (std::nothrow) woden_ctx;
    if (!ctx) return WODEN_ERR_CUDA;
    ctx->device = cuda_device;
    Bind bind(ctx);
    if (!bind.ok || cudaFree(0) != cudaSuccess) { cudaGetLastError(); delete ctx; return WODEN_ERR_CUDA; }
    *out = ctx;
    return WODEN_OK;
}

int woden_destroy(woden_ctx *ctx)
{
    if (!ctx) return WODEN_ERR_NULL;
    {
        Bind bind(ctx);
        cudaDeviceSynchronize();
        if (ctx->walk_stream) {
            cudaStreamDestroy(ctx->walk_stream);
            cudaEventDestroy(ctx->walk_fork);
            cudaEventDestroy(ctx->walk_join);
        }
        if (ctx->fit_t0) { cudaEventDestroy(ctx->fit_t0); cudaEventDestroy(ctx->fit_t1); }
        if (ctx->copy_stream) {
            cudaStreamDestroy(ctx->copy_stream);
            for (cudaEvent_t ev : ctx->chunk_done) if (ev) cudaEventDestroy(ev);
            for (cudaEvent_t ev : ctx->tile_events) cudaEventDestroy(ev);
        }
        for (DevBuf *b : {&ctx->geo, &ctx->flux, &ctx->tri, &ctx->chan, &ctx->err, &ctx->hang, &ctx->bmat, &ctx->bscale, &ctx->lut, &ctx->wblocks, &ctx->f_hx, &ctx->f_a0, &ctx->f_at, &ctx->f_small, &ctx->f_gram, &ctx->f_ops,
                          &ctx->f_part, &ctx->h_uvw, &ctx->h_comp,
                          &ctx->h_int, &ctx->h_vis})
            b->release();
    }
    delete ctx;
    return WODEN_OK;
}

const char *woden_strerror(int status)
{
    switch (status) {
    case WODEN_OK: return "ok";
    case WODEN_ERR_NULL: return "a required pointer is NULL";
    case WODEN_ERR_DIM: return "a size or scalar argument is out of range";
    case WODEN_ERR_ORDER: return "shapelet order outside 0..WODEN_MAX_ORDER";
    case WODEN_ERR_CUDA: return "CUDA error (see woden_last_error)";
    case WODEN_ERR_UNIMPLEMENTED: return "not implemented";
    case WODEN_ERR_DATA: return "device-side precondition violated (see woden_b200.h)";
    case WODEN_ERR_STATIC_LIMIT: return "size beyond the built-in scratch array of a non-allocating entry point";
    }
    return "unknown status";
}

const char *woden_last_error(const woden_ctx *ctx) { return ctx ? ctx->last_error.c_str() : ""; }

int woden_set_path(woden_ctx *ctx, int path)
{
    if (!ctx) return WODEN_ERR_NULL;
    if (path != WODEN_PATH_AUTO && path != WODEN_PATH_GENERAL) return WODEN_ERR_DIM;
    ctx->path = path;
    return WODEN_OK;
}

unsigned long long woden_kernel_launches(void) { return woden::g_kernel_launches; }

int woden_last_path(const woden_ctx *ctx) { return ctx ? ctx->last_path : WODEN_PATH_NONE; }

int woden_last_shapelet_path(const woden_ctx *ctx) { return ctx ? ctx->last_shapelet_path : WODEN_PATH_NONE; }
int woden_last_shapelet_bucket(const woden_ctx *ctx) { return ctx ? ctx->last_shapelet_bucket : -1; }

int woden_set_shapelet_path(woden_ctx *ctx, int path)
{
    if (!ctx) return WODEN_ERR_NULL;
    if (path != WODEN_SHAPELET_AUTO && path != WODEN_SHAPELET_REGISTER && path != WODEN_SHAPELET_TENSOR)
        return WODEN_ERR_DIM;
    ctx->shapelet_path = path;
    return WODEN_OK;
}

int woden_check(woden_ctx *ctx)
{
    if (!ctx) return WODEN_ERR_NULL;
    Bind bind(ctx);
    if (!bind.ok) return WODEN_ERR_CUDA;
    CU(ctx, cudaStreamSynchronize(ctx->last_stream), "woden_check sync");
    if (!ctx->err.p) return WODEN_OK;
    unsigned int n = 0;
    CU(ctx, cudaMemcpy(&n, ctx->err.p, sizeof n, cudaMemcpyDeviceToHost), "read error counter");
    CU(ctx, cudaMemset(ctx->err.p, 0, sizeof n), "clear error counter");
    return n ? WODEN_ERR_DATA : WODEN_OK;
}

int woden_predict_points(woden_ctx *ctx, const woden_uvw *uvw, int n, const double *l, const double *m,
                         const double *s0_jy, const double *alpha, double ref_freq_hz, float *vis,
                         int accumulate, void *cuda_stream)
{
    int rc = common_checks(ctx, uvw, n, l, m, s0_jy, alpha, ref_freq_hz, vis);
    if (rc != WODEN_OK) return rc;
    Bind bind(ctx);
    if (!bind.ok) return WODEN_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    ctx->last_stream = st;
    ctx->last_path = WODEN_PATH_NONE;
    if (n == 0) return zero_or_nothing(ctx, uvw, vis, accumulate, st);
    if ((rc = ensure_err(ctx, st)) != WODEN_OK) return rc;
    if ((rc = ensure_chan(ctx, uvw, st)) != WODEN_OK) return rc;
    const int n_pad = (n + KB - 1) / KB * KB;
    const bool walk = ctx->path == WODEN_PATH_AUTO && ctx->ch.uniform;
    ctx->last_path = walk ? WODEN_PATH_WALKING : WODEN_PATH_GENERAL;
    CU(ctx, ctx->geo.reserve((size_t)n_pad * sizeof(GeoP)), "alloc geometry");
    unsigned int *err = static_cast<unsigned int *>(ctx->err.p);
    launch_pack_points(l, m, n, n_pad, static_cast<GeoP *>(ctx->geo.p), err, st);
    UvwDev d{uvw->u_m, uvw->v_m, uvw->w_m, uvw->n_baselines, uvw->n_times, uvw->n_freqs};
    const GeoP *geo = static_cast<const GeoP *>(ctx->geo.p);
    float2 *out = reinterpret_cast<float2 *>(vis);
    if (walk) {
        if ((rc = ensure_walk_streams(ctx)) != WODEN_OK) return rc;
        CU(ctx, ctx->wblocks.reserve(walk_blocks_bytes(n, ctx->ch.F_pad / WALK_FT, false)), "alloc constant blocks");
        unsigned char *blocks = static_cast<unsigned char *>(ctx->wblocks.p);
        launch_pack_walk_points(geo, s0_jy, alpha, ref_freq_hz, n, ctx->ch, blocks, err, st);
        CU(ctx, cudaGetLastError(), "pack points");
        const WalkStreams ws{st, ctx->walk_stream, ctx->walk_fork, ctx->walk_join, ctx->walk_tile_done, ctx->walk_tile_user};
        CU(ctx, launch_walk_points(d, ctx->ch, blocks, n, out, accumulate ? 1 : 0, err, ws), "predict_points launch");
        return WODEN_OK;
    }
    CU(ctx, ctx->flux.reserve((size_t)ctx->ch.F_pad * n_pad * 4), "alloc flux table");
    launch_pack_flux(s0_jy, alpha, ref_freq_hz, n, n_pad, ctx->ch, PG_FT, false, static_cast<float *>(ctx->flux.p), err, st);
    CU(ctx, cudaGetLastError(), "pack points");
    CU(ctx, launch_predict_points(d, ctx->ch, geo, static_cast<const float *>(ctx->flux.p), n_pad, out,
                                  accumulate ? 1 : 0, err, st),
       "predict_points launch");
    return WODEN_OK;
}

int woden_predict_gaussians(woden_ctx *ctx, const woden_uvw *uvw, int n, const double *l, const double *m,
                            const double *s0_jy, const double *alpha, double ref_freq_hz,
                            const double *maj_fwhm_rad, const double *min_fwhm_rad, const double *pa_rad,
                            float *vis, int accumulate, void *cuda_stream)
{
    int rc = common_checks(ctx, uvw, n, l, m, s0_jy, alpha, ref_freq_hz, vis);
    if (rc != WODEN_OK) return rc;
    if (n > 0 && (!maj_fwhm_rad || !min_fwhm_rad || !pa_rad)) return WODEN_ERR_NULL;
    Bind bind(ctx);
    if (!bind.ok) return WODEN_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    ctx->last_stream = st;
    ctx->last_path = WODEN_PATH_NONE;
    if (n == 0) return zero_or_nothing(ctx, uvw, vis, accumulate, st);
    if ((rc = ensure_err(ctx, st)) != WODEN_OK) return rc;
    if ((rc = ensure_chan(ctx, uvw, st)) != WODEN_OK) return rc;
    const int n_pad = (n + KB - 1) / KB * KB;
    const bool walk = ctx->path == WODEN_PATH_AUTO && ctx->ch.uniform;
    ctx->last_path = walk ? WODEN_PATH_WALKING : WODEN_PATH_GENERAL;
    CU(ctx, ctx->geo.reserve((size_t)n_pad * sizeof(GeoG)), "alloc geometry");
    unsigned int *err = static_cast<unsigned int *>(ctx->err.p);
    launch_pack_gaussians(l, m, maj_fwhm_rad, min_fwhm_rad, pa_rad, n, n_pad, static_cast<GeoG *>(ctx->geo.p), err,
                          st);
    UvwDev d{uvw->u_m, uvw->v_m, uvw->w_m, uvw->n_baselines, uvw->n_times, uvw->n_freqs};
    const GeoG *geo = static_cast<const GeoG *>(ctx->geo.p);
    float2 *out = reinterpret_cast<float2 *>(vis);
    if (walk) {
        if ((rc = ensure_walk_streams(ctx)) != WODEN_OK) return rc;
        CU(ctx, ctx->wblocks.reserve(walk_blocks_bytes(n, ctx->ch.F_pad / WALK_FT, true)), "alloc constant blocks");
        unsigned char *blocks = static_cast<unsigned char *>(ctx->wblocks.p);
        launch_pack_walk_gaussians(geo, s0_jy, alpha, ref_freq_hz, n, ctx->ch, blocks, err, st);
        CU(ctx, cudaGetLastError(), "pack gaussians");
        const WalkStreams ws{st, ctx->walk_stream, ctx->walk_fork, ctx->walk_join, ctx->walk_tile_done, ctx->walk_tile_user};
        CU(ctx, launch_walk_gaussians(d, ctx->ch, blocks, n, out, accumulate ? 1 : 0, err, ws),
           "predict_gaussians launch");
        return WODEN_OK;
    }
    CU(ctx, ctx->flux.reserve((size_t)ctx->ch.F_pad * n_pad * 4), "alloc flux table");
    launch_pack_flux(s0_jy, alpha, ref_freq_hz, n, n_pad, ctx->ch, PG_FT, false, static_cast<float *>(ctx->flux.p), err, st);
    CU(ctx, cudaGetLastError(), "pack gaussians");
    CU(ctx, launch_predict_gaussians(d, ctx->ch, geo, static_cast<const float *>(ctx->flux.p), n_pad, out,
                                     accumulate ? 1 : 0, err, st),
       "predict_gaussians launch");
    return WODEN_OK;
}

int woden_predict_shapelets(woden_ctx *ctx, const woden_uvw *uvw, int n, const double *l, const double *m,
                            const double *s0_jy, const double *alpha, double ref_freq_hz,
                            const double *beta1_rad, const double *beta2_rad, const double *pa_rad,
                            const double *uv_basis, const int *coeff_offset, int n_coeff, int p_max,
                            const int *n1, const int *n2, const double *coeff, float *vis, int accumulate,
                            void *cuda_stream)
{
    int rc = common_checks(ctx, uvw, n, l, m, s0_jy, alpha, ref_freq_hz, vis);
    if (rc != WODEN_OK) return rc;
    if (n > 0 && (!beta1_rad || !beta2_rad || !pa_rad || !coeff_offset)) return WODEN_ERR_NULL;
    if (n_coeff < 0) return WODEN_ERR_DIM;
    if (n_coeff > 0 && (!n1 || !n2 || !coeff)) return WODEN_ERR_NULL;
    if (p_max < 0 || p_max > WODEN_MAX_ORDER) return WODEN_ERR_ORDER;
    Bind bind(ctx);
    if (!bind.ok) return WODEN_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    ctx->last_stream = st;
    ctx->last_shapelet_path = WODEN_PATH_NONE;
    ctx->last_shapelet_bucket = -1;
    if (n == 0) return zero_or_nothing(ctx, uvw, vis, accumulate, st);
    if ((rc = ensure_err(ctx, st)) != WODEN_OK) return rc;
    if ((rc = ensure_chan(ctx, uvw, st)) != WODEN_OK) return rc;
    // compile-time order bucket PM >= p_max; pack_coeffs flags any (n1, n2) with n1 + n2 > p_max
    int PM = shapelet_order_bucket(p_max);
    if (PM < 0) return WODEN_ERR_ORDER;
    const size_t tri_floats = (size_t)tri_stride(PM);
    CU(ctx, ctx->geo.reserve((size_t)n * sizeof(GeoS)), "alloc geometry");
    CU(ctx, ctx->tri.reserve((size_t)n * tri_floats * 4), "alloc coefficient triangles");
    CU(ctx, ctx->flux.reserve((size_t)ctx->ch.F_pad * n * 4), "alloc flux table");
    unsigned int *err = static_cast<unsigned int *>(ctx->err.p);
    launch_pack_shapelets(l, m, beta1_rad, beta2_rad, pa_rad, uv_basis, n, PM, static_cast<GeoS *>(ctx->geo.p), err,
                          st);
    launch_pack_coeffs(coeff_offset, n1, n2, coeff, n, n_coeff, p_max, PM, static_cast<float *>(ctx->tri.p), err, st);
    launch_pack_flux(s0_jy, alpha, ref_freq_hz, n, n, ctx->ch, SH_FT, false, static_cast<float *>(ctx->flux.p), err, st);
    CU(ctx, cudaGetLastError(), "pack shapelets");
    UvwDev d{uvw->u_m, uvw->v_m, uvw->w_m, uvw->n_baselines, uvw->n_times, uvw->n_freqs};
    // truncated models: when under 3/4 of the order bucket's triangle is listed, take
    // the kernel variant that skips empty 4-coefficient chunks (decided from the list length alone)
    const bool sparse = (double)n_coeff < 0.75 * (double)n * (double)((PM + 1) * (PM + 2) / 2);
    // tensor-core variant (north_star: "used only if ... shown by measurement to beat the register path"):
    // AUTO takes it from the order bucket at which it measured faster (profiles/shapelet_mma_r2.md)
    const bool tensor = ctx->shapelet_path == WODEN_SHAPELET_TENSOR ||
                        (ctx->shapelet_path == WODEN_SHAPELET_AUTO && PM >= SHAPELET_TENSOR_MIN_ORDER);
    ctx->last_shapelet_bucket = PM;
    ctx->last_shapelet_path = tensor ? WODEN_SHAPELET_TENSOR : sparse ? WODEN_SHAPELET_REGISTER_SPARSE : WODEN_SHAPELET_REGISTER;
    if (tensor) {
        CU(ctx, ctx->bmat.reserve(mma_bmat_halves(PM, n) * 2), "alloc coefficient matrices");
        CU(ctx, ctx->bscale.reserve((size_t)n * 4), "alloc coefficient scales");
        CU(ctx, launch_predict_shapelets_mma(d, ctx->ch, static_cast<const GeoS *>(ctx->geo.p),
                                             static_cast<const float *>(ctx->tri.p),
                                             static_cast<const float *>(ctx->flux.p), n, PM,
                                             static_cast<__half *>(ctx->bmat.p), static_cast<float *>(ctx->bscale.p),
                                             reinterpret_cast<float2 *>(vis), accumulate ? 1 : 0, st),
           "predict_shapelets (tensor) launch");
        return WODEN_OK;
    }
    CU(ctx, launch_predict_shapelets(d, ctx->ch, static_cast<const GeoS *>(ctx->geo.p),
                                     static_cast<const float *>(ctx->tri.p),
                                     static_cast<const float *>(ctx->flux.p), n, PM, sparse,
                                     reinterpret_cast<float2 *>(vis), accumulate ? 1 : 0, st),
       "predict_shapelets launch");
    return WODEN_OK;
}

}  // extern "C"

namespace {

// sequential sub-allocation of one device arena, 256-byte aligned
struct Arena {
    char *base;
    size_t off = 0;
    explicit Arena(void *p) : base(static_cast<char *>(p)) {}
    static size_t pad(size_t b) { return (b + 255) & ~(size_t)255; }
    template <typename T>
    T *put(woden_ctx *ctx, const T *host, size_t count, cudaStream_t st, cudaError_t *e)
    {
        if (!host || count == 0) return nullptr;
        T *dst = reinterpret_cast<T *>(base + off);
        off += pad(count * sizeof(T));
        if (*e == cudaSuccess) *e = cudaMemcpyAsync(dst, host, count * sizeof(T), cudaMemcpyHostToDevice, st);
        (void)ctx;
        return dst;
    }
};

}  // namespace

extern "C" {

int woden_simulate_host(woden_ctx *ctx, int n_baselines, int n_times, int n_freqs, const double *u_m,
                        const double *v_m, const double *w_m, const double *freqs_hz, double ref_freq_hz,
                        const woden_points_host *pts, const woden_gaussians_host *gau,
                        const woden_shapelets_host *shp, float *vis_host, void *cuda_stream)
{
    if (!ctx || !u_m || !v_m || !w_m || !freqs_hz || !vis_host) return WODEN_ERR_NULL;
    if (n_baselines <= 0 || n_times <= 0 || n_freqs <= 0) return WODEN_ERR_DIM;
    const int np = pts ? pts->n : 0, ng = gau ? gau->n : 0, ns = shp ? shp->n : 0;
    if (np < 0 || ng < 0 || ns < 0) return WODEN_ERR_DIM;
    if (np > 0 && (!pts->l || !pts->m || !pts->s0_jy || !pts->alpha)) return WODEN_ERR_NULL;
    if (ng > 0 && (!gau->l || !gau->m || !gau->s0_jy || !gau->alpha || !gau->maj_fwhm_rad || !gau->min_fwhm_rad ||
                   !gau->pa_rad))
        return WODEN_ERR_NULL;
    if (ns > 0) {
        if (!shp->l || !shp->m || !shp->s0_jy || !shp->alpha || !shp->beta1_rad || !shp->beta2_rad || !shp->pa_rad ||
            !shp->coeff_offset)
            return WODEN_ERR_NULL;
        if (shp->n_coeff < 0) return WODEN_ERR_DIM;
        if (shp->n_coeff > 0 && (!shp->n1 || !shp->n2 || !shp->coeff)) return WODEN_ERR_NULL;
        if (shp->coeff_offset[ns] != shp->n_coeff) return WODEN_ERR_DIM;
    }
    Bind bind(ctx);
    if (!bind.ok) return WODEN_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const size_t TB = (size_t)n_times * n_baselines;
    const size_t nvis = TB * n_freqs;
    const size_t nc = ns > 0 ? (size_t)shp->n_coeff : 0;
    size_t comp_bytes = Arena::pad(8 * (size_t)np) * 4 + Arena::pad(8 * (size_t)ng) * 7 +
                        Arena::pad(8 * (size_t)ns) * 7 + Arena::pad(48 * (size_t)ns) + Arena::pad(8 * nc) +
                        Arena::pad(4 * ((size_t)ns + 1)) + 2 * Arena::pad(4 * nc) + 4096;
    CU(ctx, ctx->h_uvw.reserve(3 * Arena::pad(TB * 8)), "alloc uvw");
    CU(ctx, ctx->h_comp.reserve(comp_bytes), "alloc components");
    CU(ctx, ctx->h_vis.reserve(nvis * 8), "alloc vis");
    cudaError_t e = cudaSuccess;
    Arena au(ctx->h_uvw.p), ac(ctx->h_comp.p);
    woden_uvw uvw;
    uvw.n_baselines = n_baselines; uvw.n_times = n_times; uvw.n_freqs = n_freqs;
    uvw.u_m = au.put(ctx, u_m, TB, st, &e);
    uvw.v_m = au.put(ctx, v_m, TB, st, &e);
    uvw.w_m = au.put(ctx, w_m, TB, st, &e);
    uvw.freqs_hz = freqs_hz;
    float *vis = static_cast<float *>(ctx->h_vis.p);

    const double *pl = nullptr, *pm = nullptr, *ps = nullptr, *pa = nullptr;
    if (np > 0) {
        pl = ac.put(ctx, pts->l, np, st, &e); pm = ac.put(ctx, pts->m, np, st, &e);
        ps = ac.put(ctx, pts->s0_jy, np, st, &e); pa = ac.put(ctx, pts->alpha, np, st, &e);
    }
    const double *gl = nullptr, *gm = nullptr, *gs = nullptr, *ga = nullptr, *gmj = nullptr, *gmn = nullptr,
                 *gpa = nullptr;
    if (ng > 0) {
        gl = ac.put(ctx, gau->l, ng, st, &e); gm = ac.put(ctx, gau->m, ng, st, &e);
        gs = ac.put(ctx, gau->s0_jy, ng, st, &e); ga = ac.put(ctx, gau->alpha, ng, st, &e);
        gmj = ac.put(ctx, gau->maj_fwhm_rad, ng, st, &e); gmn = ac.put(ctx, gau->min_fwhm_rad, ng, st, &e);
        gpa = ac.put(ctx, gau->pa_rad, ng, st, &e);
    }
    const double *sl = nullptr, *sm = nullptr, *ss = nullptr, *sa = nullptr, *sb1 = nullptr, *sb2 = nullptr,
                 *spa = nullptr, *sM = nullptr, *sc = nullptr;
    const int *so = nullptr, *sn1 = nullptr, *sn2 = nullptr;
    if (ns > 0) {
        sl = ac.put(ctx, shp->l, ns, st, &e); sm = ac.put(ctx, shp->m, ns, st, &e);
        ss = ac.put(ctx, shp->s0_jy, ns, st, &e); sa = ac.put(ctx, shp->alpha, ns, st, &e);
        sb1 = ac.put(ctx, shp->beta1_rad, ns, st, &e); sb2 = ac.put(ctx, shp->beta2_rad, ns, st, &e);
        spa = ac.put(ctx, shp->pa_rad, ns, st, &e);
        sM = ac.put(ctx, shp->uv_basis, (size_t)6 * ns, st, &e);
        sc = ac.put(ctx, shp->coeff, nc, st, &e);
        so = ac.put(ctx, shp->coeff_offset, (size_t)ns + 1, st, &e);
        sn1 = ac.put(ctx, shp->n1, nc, st, &e); sn2 = ac.put(ctx, shp->n2, nc, st, &e);
    }
    if (e != cudaSuccess) return fail_cuda(ctx, e, "host->device copies");

    // Order of the three types: shapelets (overwrite), points, Gaussians -- the first non-empty type overwrites
    // the buffer, the others accumulate.  The device-to-host copy (PCIe: ~28 ms for config 5's 1.4 GB) hides
    // behind the LAST predictor:
    //  * channel-walking path, >= 2 channel tiles: the last type (Gaussians, else points) finishes the
    //    output one 32-channel tile at a time; each finished tile is copied back (a strided 2-D copy) on a
    //    second stream while the following tiles are computed.  Only the last tile's copy is exposed.
    //  * otherwise: time steps are independent (Eq 9 sums over components only), so the last predictor runs in
    //    chunks of time steps and each finished chunk is copied back meanwhile.
    if (!ctx->copy_stream) {
        CU(ctx, cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking), "create copy stream");
        for (cudaEvent_t &ev : ctx->chunk_done) CU(ctx, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming), "create event");
    }
    int rc = ensure_chan(ctx, &uvw, st);
    if (rc != WODEN_OK) return rc;
    const int last = ng > 0 ? 1 : (np > 0 ? 0 : (ns > 0 ? 2 : 0));     // 0 points, 1 Gaussians, 2 shapelets
    const int n_ftiles = ctx->ch.F_pad / WALK_FT;
    // a copy into pageable memory blocks the HOST until it is done: issued from the launch loop it would starve the
    // GPU of the launches that follow, so only page-locked buffers take the tile-wise path
    cudaPointerAttributes attr;
    const bool pinned = cudaPointerGetAttributes(&attr, vis_host) == cudaSuccess && attr.type == cudaMemoryTypeHost;
    cudaGetLastError();
    const bool by_tile = pinned && last != 2 && ctx->path == WODEN_PATH_AUTO && ctx->ch.uniform && n_ftiles >= 2;
    int written = 0;
    if (last != 2 && ns > 0) {
        rc = woden_predict_shapelets(ctx, &uvw, ns, sl, sm, ss, sa, ref_freq_hz, sb1, sb2, spa, sM, so, (int)nc,
                                     shp->p_max, sn1, sn2, sc, vis, 0, st);
        written = 1;
    }
    if (rc == WODEN_OK && last == 1 && np > 0) {
        rc = woden_predict_points(ctx, &uvw, np, pl, pm, ps, pa, ref_freq_hz, vis, written, st);
        written = 1;
    }
    if (rc == WODEN_OK && by_tile) {
        struct TileCopy {
            woden_ctx *ctx; const float *vis; float *vis_host; int T, F, B; cudaError_t err; int calls;
        } tc{ctx, vis, vis_host, n_times, n_freqs, n_baselines, cudaSuccess, 0};
        while ((int)ctx->tile_events.size() < n_ftiles) {
            cudaEvent_t ev;
            CU(ctx, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming), "create event");
            ctx->tile_events.push_back(ev);
        }
        ctx->walk_tile_user = &tc;
        ctx->walk_tile_done = [](void *user, int ftile, cudaStream_t s) {
            TileCopy *t = static_cast<TileCopy *>(user);
            ++t->calls;
            const int f0 = ftile * WALK_FT, nf = t->F - f0 < WALK_FT ? t->F - f0 : WALK_FT;
            if (nf <= 0 || t->err != cudaSuccess) return;
            cudaEvent_t ev = t->ctx->tile_events[ftile];
            cudaError_t e = cudaEventRecord(ev, s);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(t->ctx->copy_stream, ev, 0);
            const size_t pitch = (size_t)t->F * t->B * 8, off = (size_t)f0 * t->B * 2;
            if (e == cudaSuccess)
                e = cudaMemcpy2DAsync(t->vis_host + off, pitch, t->vis + off, pitch, (size_t)nf * t->B * 8, t->T,
                                      cudaMemcpyDeviceToHost, t->ctx->copy_stream);
            t->err = e;
        };
        if (last == 1)
            rc = woden_predict_gaussians(ctx, &uvw, ng, gl, gm, gs, ga, ref_freq_hz, gmj, gmn, gpa, vis, written, st);
        else
            rc = woden_predict_points(ctx, &uvw, np, pl, pm, ps, pa, ref_freq_hz, vis, written, st);
        ctx->walk_tile_done = nullptr;
        ctx->walk_tile_user = nullptr;
        if (rc == WODEN_OK && tc.err != cudaSuccess) rc = fail_cuda(ctx, tc.err, "device->host vis (tile)");
        if (rc == WODEN_OK && tc.calls != n_ftiles) {      // the call did not take the tile-wise path after all
            CU(ctx, cudaEventRecord(ctx->chunk_done[0], st), "record");
            CU(ctx, cudaStreamWaitEvent(ctx->copy_stream, ctx->chunk_done[0], 0), "wait");
            CU(ctx, cudaMemcpyAsync(vis_host, vis, nvis * 8, cudaMemcpyDeviceToHost, ctx->copy_stream), "device->host vis");
        }
    } else if (rc == WODEN_OK) {
        // chunks of >= 64 MB of output: enough to hide the copy-back, not so many that the last predictor's
        // launch sequence (staging included) is repeated over small grids
        int n_chunks = (int)((nvis * 8 + (64u << 20) - 1) / (64u << 20));
        if (n_chunks > SIM_CHUNKS) n_chunks = SIM_CHUNKS;
        if (n_chunks > n_times) n_chunks = n_times;
        if (n_chunks < 1) n_chunks = 1;
        for (int c = 0; c < n_chunks && rc == WODEN_OK; ++c) {
            const int t0 = (int)((long long)n_times * c / n_chunks), t1 = (int)((long long)n_times * (c + 1) / n_chunks);
            woden_uvw part = uvw;
            part.n_times = t1 - t0;
            part.u_m = uvw.u_m + (size_t)t0 * n_baselines;
            part.v_m = uvw.v_m + (size_t)t0 * n_baselines;
            part.w_m = uvw.w_m + (size_t)t0 * n_baselines;
            const size_t off = (size_t)t0 * n_freqs * n_baselines, cnt = (size_t)(t1 - t0) * n_freqs * n_baselines;
            float *vc = vis + 2 * off;
            if (last == 0)
                rc = woden_predict_points(ctx, &part, np, pl, pm, ps, pa, ref_freq_hz, vc, written, st);
            else if (last == 1)
                rc = woden_predict_gaussians(ctx, &part, ng, gl, gm, gs, ga, ref_freq_hz, gmj, gmn, gpa, vc, written, st);
            else
                rc = woden_predict_shapelets(ctx, &part, ns, sl, sm, ss, sa, ref_freq_hz, sb1, sb2, spa, sM, so, (int)nc,
                                             shp ? shp->p_max : 0, sn1, sn2, sc, vc, 0, st);
            if (rc != WODEN_OK) break;
            CU(ctx, cudaEventRecord(ctx->chunk_done[c], st), "record chunk");
            CU(ctx, cudaStreamWaitEvent(ctx->copy_stream, ctx->chunk_done[c], 0), "wait chunk");
            CU(ctx, cudaMemcpyAsync(vis_host + 2 * off, vc, cnt * 8, cudaMemcpyDeviceToHost, ctx->copy_stream),
               "device->host vis");
        }
    }
    if (rc != WODEN_OK) { cudaStreamSynchronize(st); cudaStreamSynchronize(ctx->copy_stream); return rc; }
    CU(ctx, cudaStreamSynchronize(st), "simulate sync");
    CU(ctx, cudaStreamSynchronize(ctx->copy_stream), "simulate copy sync");
    ctx->last_stream = st;
    return WODEN_OK;
}

int woden_uvw_from_antennas(woden_ctx *ctx, int n_antennas, const double *x_m, const double *y_m, const double *z_m,
                            int n_times, const double *hour_angle_rad, double dec0_rad, double *u_m, double *v_m,
                            double *w_m, void *cuda_stream)
{
    if (!ctx || !x_m || !y_m || !z_m || !hour_angle_rad || !u_m || !v_m || !w_m) return WODEN_ERR_NULL;
    if (n_antennas < 2 || n_antennas > 46340 || n_times <= 0 || !std::isfinite(dec0_rad)) return WODEN_ERR_DIM;
    for (int t = 0; t < n_times; ++t)
        if (!std::isfinite(hour_angle_rad[t])) return WODEN_ERR_DIM;
    Bind bind(ctx);
    if (!bind.ok) return WODEN_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    ctx->last_stream = st;
    CU(ctx, ctx->hang.reserve((size_t)n_times * 8), "alloc hour angles");
    // pageable source: staged by the runtime before the call returns
    CU(ctx, cudaMemcpyAsync(ctx->hang.p, hour_angle_rad, (size_t)n_times * 8, cudaMemcpyHostToDevice, st),
       "upload hour angles");
    CU(ctx, launch_uvw(x_m, y_m, z_m, n_antennas, n_times, static_cast<const double *>(ctx->hang.p), dec0_rad, u_m, v_m,
                       w_m, st),
       "uvw launch");
    return WODEN_OK;
}

int woden_shapelet_uv_basis(woden_ctx *ctx, int n, const double *l, const double *m, double dec0_rad,
                            double *uv_basis, void *cuda_stream)
{
    if (!ctx) return WODEN_ERR_NULL;
    if (n < 0 || !std::isfinite(dec0_rad)) return WODEN_ERR_DIM;
    if (n == 0) return WODEN_OK;
    if (!l || !m || !uv_basis) return WODEN_ERR_NULL;
    Bind bind(ctx);
    if (!bind.ok) return WODEN_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    ctx->last_stream = st;
    int rc = ensure_err(ctx, st);
    if (rc != WODEN_OK) return rc;
    CU(ctx, launch_uv_basis(l, m, n, dec0_rad, uv_basis, static_cast<unsigned int *>(ctx->err.p), st),
       "uv_basis launch");
    return WODEN_OK;
}

int woden_calibrate_gains(woden_ctx *ctx, int n_antennas, long long n_cells, const float *vis_data,
                          const float *vis_model, int n_iter, double *gains, void *cuda_stream)
{
    if (!ctx || !vis_data || !vis_model || !gains) return WODEN_ERR_NULL;
    if (n_antennas < 2 || n_cells <= 0 || n_cells > 2147483647LL || n_iter < 0) return WODEN_ERR_DIM;
    if (n_antennas > 200 || calibrate_smem_bytes(n_antennas) > 227u * 1024u) return WODEN_ERR_DIM;   // W must fit shared memory
    Bind bind(ctx);
    if (!bind.ok) return WODEN_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    ctx->last_stream = st;
    CU(ctx, launch_calibrate(reinterpret_cast<const float2 *>(vis_data), reinterpret_cast<const float2 *>(vis_model),
                             reinterpret_cast<double2 *>(gains), n_antennas, n_cells, n_iter, st),
       "calibrate launch");
    return WODEN_OK;
}

int woden_peel(woden_ctx *ctx, int n_antennas, long long n_cells, const float *vis_data, const float *vis_model,
               const double *gains, float *vis_out, void *cuda_stream)
{
    if (!ctx || !vis_data || !vis_model || !gains || !vis_out) return WODEN_ERR_NULL;
    if (n_antennas < 2 || n_antennas > 3000 || n_cells <= 0 || n_cells > 2147483647LL) return WODEN_ERR_DIM;
    Bind bind(ctx);
    if (!bind.ok) return WODEN_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    ctx->last_stream = st;
    CU(ctx, launch_peel(reinterpret_cast<const float2 *>(vis_data), reinterpret_cast<const float2 *>(vis_model),
                        reinterpret_cast<const double2 *>(gains), reinterpret_cast<float2 *>(vis_out), n_antennas,
                        n_cells, st),
       "peel launch");
    return WODEN_OK;
}

}  // extern "C"

namespace {

// argument checks and scratch of the image-space entry points; `full` also allocates the solver's buffers
int fit_setup(woden_ctx *ctx, const woden_image_grid *grid, double l0, double m0, double pa_rad, int p_max,
              const woden_restoring_beam *beam, bool full, cudaStream_t st, FitScratch *w, FitProblem *f, FitSizes *szo)
{
    if (p_max < 0 || p_max > (full ? WODEN_FIT_MAX_ORDER : WODEN_MAX_ORDER)) return WODEN_ERR_ORDER;
    if (grid->n_l <= 0 || grid->n_m <= 0 || (long long)grid->n_l * grid->n_m > (1LL << 22) || !(grid->dl != 0.0) ||
        !(grid->dm != 0.0) || !std::isfinite(grid->dl) || !std::isfinite(grid->dm) || !std::isfinite(grid->l_c) ||
        !std::isfinite(grid->m_c) || !std::isfinite(l0) || !std::isfinite(m0) || !std::isfinite(pa_rad))
        return WODEN_ERR_DIM;
    const bool has_beam = beam && beam->bmaj_rad > 0.0;
    if (has_beam && (beam->half_width < 0 || beam->half_width > 24 || !(beam->bmin_rad >= 0.0) ||
                     !std::isfinite(beam->bmaj_rad) || !std::isfinite(beam->bmin_rad) || !std::isfinite(beam->bpa_rad)))
        return WODEN_ERR_DIM;
    int rc = ensure_err(ctx, st);
    if (rc != WODEN_OK) return rc;
    const int n_pix = grid->n_l * grid->n_m;
    const FitSizes sz = fit_sizes(n_pix, p_max);
    if (full && sz.n_pad > FIT_MAX_N) return WODEN_ERR_ORDER;
    if (sz.at_doubles > (1ull << 32)) return WODEN_ERR_DIM;             // 32 GB of FP64 design matrix
    const size_t small = (size_t)4 * sz.n_pad + n_pix + 49 * 49 + 64;        // scale, abssum, z, g | r | stencil
    CU(ctx, ctx->f_hx.reserve(sz.hermite_doubles * 8), "alloc fit Hermite tables");
    CU(ctx, ctx->f_at.reserve(sz.at_doubles * 8), "alloc fit design matrix");
    if (has_beam) CU(ctx, ctx->f_a0.reserve(sz.at_doubles * 8), "alloc fit unconvolved basis");
    CU(ctx, ctx->f_small.reserve(small * 8), "alloc fit vectors");
    if (full) {
        CU(ctx, ctx->f_gram.reserve(sz.gram_doubles * 8), "alloc fit Gram matrix");
        CU(ctx, ctx->f_ops.reserve(sz.ops_halves * 2), "alloc fit operands");
        CU(ctx, ctx->f_part.reserve(sz.partial_floats * 4), "alloc fit partials");
        if (!ctx->fit_t0) {
            CU(ctx, cudaEventCreate(&ctx->fit_t0), "create event");
            CU(ctx, cudaEventCreate(&ctx->fit_t1), "create event");
        }
    }
    w->hx = static_cast<double *>(ctx->f_hx.p);
    w->a0 = static_cast<double *>(ctx->f_a0.p);
    w->at = static_cast<double *>(ctx->f_at.p);
    double *v = static_cast<double *>(ctx->f_small.p);
    w->scale = v; w->abssum = v + sz.n_pad; w->z = v + 2 * sz.n_pad; w->g = v + 3 * sz.n_pad;
    w->r = v + 4 * sz.n_pad; w->stencil = w->r + n_pix;
    w->gram = static_cast<double *>(ctx->f_gram.p);
    w->ops = static_cast<__half *>(ctx->f_ops.p);
    w->partial = static_cast<float *>(ctx->f_part.p);
    w->err = static_cast<unsigned int *>(ctx->err.p);
    w->gram_t0 = full ? ctx->fit_t0 : nullptr; w->gram_t1 = full ? ctx->fit_t1 : nullptr;
    f->n_l = grid->n_l; f->n_m = grid->n_m; f->p_max = p_max;
    f->half_width = has_beam ? beam->half_width : 0;
    f->n_refine = 0;
    f->dl = grid->dl; f->dm = grid->dm; f->l_c = grid->l_c; f->m_c = grid->m_c; f->l0 = l0; f->m0 = m0; f->pa = pa_rad;
    f->bmaj = has_beam ? beam->bmaj_rad : 0.0; f->bmin = has_beam ? beam->bmin_rad : 0.0; f->bpa = has_beam ? beam->bpa_rad : 0.0;
    f->image = nullptr; f->coeff = nullptr; f->weights = nullptr; f->residual = nullptr;
    *szo = sz;
    return WODEN_OK;
}

}  // namespace

extern "C" {

int woden_fit_shapelets(woden_ctx *ctx, const woden_image_grid *grid, const double *image, double l0, double m0,
                        double pa_rad, int p_max, int n_beta, const double *beta1_rad, const double *beta2_rad,
                        const woden_restoring_beam *beam, int n_refine, double *coeff, double *residual,
                        double *weights, int *best, void *cuda_stream)
{
    if (!ctx || !grid || !image || !beta1_rad || !beta2_rad || !coeff || !residual) return WODEN_ERR_NULL;
    if (n_beta <= 0 || n_refine < 0) return WODEN_ERR_DIM;
    for (int k = 0; k < n_beta; ++k)
        if (!(beta1_rad[k] > 0.0) || !(beta2_rad[k] > 0.0) || !std::isfinite(beta1_rad[k]) || !std::isfinite(beta2_rad[k]))
            return WODEN_ERR_DIM;
    Bind bind(ctx);
    if (!bind.ok) return WODEN_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    ctx->last_stream = st;
    FitScratch w;
    FitProblem f;
    FitSizes sz;
    int rc = fit_setup(ctx, grid, l0, m0, pa_rad, p_max, beam, true, st, &w, &f, &sz);
    if (rc != WODEN_OK) return rc;
    f.n_refine = n_refine > 0 ? n_refine : 6;
    f.image = image;
    for (int k = 0; k < n_beta; ++k) {
        f.beta1 = beta1_rad[k]; f.beta2 = beta2_rad[k];
        f.coeff = coeff + (size_t)k * sz.P;
        f.weights = weights ? weights + (size_t)k * sz.P : nullptr;
        f.residual = residual + k;
        CU(ctx, launch_fit_one(f, w, st), "fit launch");
    }
    if (best) CU(ctx, launch_fit_argmin(residual, n_beta, best, st), "fit argmin launch");
    return WODEN_OK;
}

int woden_shapelet_basis_sums(woden_ctx *ctx, const woden_image_grid *grid, double l0, double m0, double pa_rad, int p_max,
                              double beta1_rad, double beta2_rad, const woden_restoring_beam *beam, double *abs_sums,
                              void *cuda_stream)
{
    if (!ctx || !grid || !abs_sums) return WODEN_ERR_NULL;
    if (!(beta1_rad > 0.0) || !(beta2_rad > 0.0) || !std::isfinite(beta1_rad) || !std::isfinite(beta2_rad)) return WODEN_ERR_DIM;
    Bind bind(ctx);
    if (!bind.ok) return WODEN_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    ctx->last_stream = st;
    FitScratch w;
    FitProblem f;
    FitSizes sz;
    int rc = fit_setup(ctx, grid, l0, m0, pa_rad, p_max, beam, false, st, &w, &f, &sz);
    if (rc != WODEN_OK) return rc;
    f.beta1 = beta1_rad; f.beta2 = beta2_rad;
    CU(ctx, launch_fit_basis_sums(f, w, abs_sums, st), "basis sums launch");
    return WODEN_OK;
}

int woden_shapelet_truncation_weights(woden_ctx *ctx, int n, const double *s0_jy, const double *beta1_rad,
                                      const double *beta2_rad, const double *pa_rad, const int *coeff_offset,
                                      const int *n1, const int *n2, const double *coeff, int n_pix,
                                      double beam_fwhm_rad, double *weights, void *cuda_stream)
{
    if (!ctx) return WODEN_ERR_NULL;
    if (n < 0) return WODEN_ERR_DIM;
    if (n == 0) return WODEN_OK;
    if (!s0_jy || !beta1_rad || !beta2_rad || !pa_rad || !coeff_offset) return WODEN_ERR_NULL;
    const int n_coeff = coeff_offset[n];
    if (coeff_offset[0] != 0 || n_coeff < 0) return WODEN_ERR_DIM;
    for (int j = 0; j < n; ++j)
        if (coeff_offset[j + 1] < coeff_offset[j]) return WODEN_ERR_DIM;
    if (n_coeff == 0) return WODEN_OK;
    if (!n1 || !n2 || !coeff || !weights) return WODEN_ERR_NULL;
    if (n_pix <= 0) n_pix = WODEN_EQ25_PIXELS;
    if (beam_fwhm_rad < 0.0) beam_fwhm_rad = WODEN_EQ25_BEAM_FWHM_RAD;
    if (n_pix < 3 || n_pix > 2048 || !std::isfinite(beam_fwhm_rad)) return WODEN_ERR_DIM;
    Bind bind(ctx);
    if (!bind.ok) return WODEN_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    ctx->last_stream = st;
    int rc = ensure_err(ctx, st);
    if (rc != WODEN_OK) return rc;
    // the coefficient lists go to the device once (pageable source: staged by the runtime before the call returns)
    const size_t ints = ((size_t)n_coeff * sizeof(int) + 7) / 8 * 8;
    CU(ctx, ctx->t_list.reserve(2 * ints + (size_t)n_coeff * sizeof(double)), "alloc coefficient lists");
    unsigned char *base = static_cast<unsigned char *>(ctx->t_list.p);
    int *d_n1 = reinterpret_cast<int *>(base), *d_n2 = reinterpret_cast<int *>(base + ints);
    double *d_cf = reinterpret_cast<double *>(base + 2 * ints);
    CU(ctx, cudaMemcpyAsync(d_n1, n1, (size_t)n_coeff * sizeof(int), cudaMemcpyHostToDevice, st), "upload n1");
    CU(ctx, cudaMemcpyAsync(d_n2, n2, (size_t)n_coeff * sizeof(int), cudaMemcpyHostToDevice, st), "upload n2");
    CU(ctx, cudaMemcpyAsync(d_cf, coeff, (size_t)n_coeff * sizeof(double), cudaMemcpyHostToDevice, st), "upload coefficients");
    const double a = 2.0 * std::sqrt(2.0 * std::log(2.0));
    for (int j = 0; j < n; ++j) {
        const int lo = coeff_offset[j], hi = coeff_offset[j + 1];
        if (hi == lo) continue;
        int pm = 0;
        for (int i = lo; i < hi; ++i) {
            if (n1[i] < 0 || n2[i] < 0 || n1[i] + n2[i] > WODEN_MAX_ORDER) return WODEN_ERR_ORDER;
            pm = std::max(pm, n1[i] + n2[i]);
        }
        if (!(beta1_rad[j] > 0.0) || !(beta2_rad[j] > 0.0) || !std::isfinite(beta1_rad[j]) || !std::isfinite(beta2_rad[j]))
            return WODEN_ERR_DIM;
        // reading G20: n_pix^2 pixels over +-1.5 sqrt(2 pm + 1) max(beta) / a per axis, centred on the component
        const double half = 1.5 * std::sqrt(2.0 * pm + 1.0) * std::max(beta1_rad[j], beta2_rad[j]) / a;
        const double pix = 2.0 * half / (n_pix - 1);
        woden_image_grid grid{n_pix, n_pix, -pix, pix, 0.0, 0.0};
        woden_restoring_beam beam{beam_fwhm_rad, beam_fwhm_rad, 0.0, 0};
        if (beam_fwhm_rad > 0.0) beam.half_width = (int)std::min(24.0, std::ceil(1.5 * beam_fwhm_rad / pix));
        FitScratch w;
        FitProblem f;
        FitSizes sz;
        rc = fit_setup(ctx, &grid, 0.0, 0.0, pa_rad[j], pm, beam_fwhm_rad > 0.0 ? &beam : nullptr, false, st, &w, &f, &sz);
        if (rc != WODEN_OK) return rc;
        f.beta1 = beta1_rad[j]; f.beta2 = beta2_rad[j];
        const int P = (pm + 1) * (pm + 2) / 2;
        CU(ctx, ctx->t_sums.reserve((size_t)P * sizeof(double)), "alloc basis sums");
        double *sums = static_cast<double *>(ctx->t_sums.p);
        CU(ctx, launch_fit_basis_sums(f, w, sums, st), "basis sums launch");
        CU(ctx, launch_eq25_weights(d_cf + lo, d_n1 + lo, d_n2 + lo, hi - lo, pm, s0_jy[j], sums, weights + lo,
                                    static_cast<unsigned int *>(ctx->err.p), st), "Eq 25 weights launch");
    }
    return WODEN_OK;
}

int woden_truncate_select(woden_ctx *ctx, int n, const double *weights, double f_comp, int *keep, int *n_keep, void *cuda_stream)
{
    if (!ctx) return WODEN_ERR_NULL;
    if (n < 0 || n > (1 << 17) || !(f_comp >= 0.0)) return WODEN_ERR_DIM;
    if (!n_keep || (n > 0 && (!weights || !keep))) return WODEN_ERR_NULL;
    Bind bind(ctx);
    if (!bind.ok) return WODEN_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    ctx->last_stream = st;
    if (n == 0) { CU(ctx, cudaMemsetAsync(n_keep, 0, sizeof(int), st), "truncate zero"); return WODEN_OK; }
    int rc = ensure_err(ctx, st);
    if (rc != WODEN_OK) return rc;
    CU(ctx, ctx->f_small.reserve((size_t)n * 12 + 64), "alloc truncation scratch");
    double *sorted = static_cast<double *>(ctx->f_small.p);
    int *rank = reinterpret_cast<int *>(sorted + n);
    CU(ctx, launch_truncate_select(weights, n, f_comp, rank, sorted, keep, n_keep,
                                   static_cast<unsigned int *>(ctx->err.p), st), "truncate launch");
    return WODEN_OK;
}

int woden_fit_gram_ms(woden_ctx *ctx, float *ms)
{
    if (!ctx || !ms) return WODEN_ERR_NULL;
    if (!ctx->fit_t0) return WODEN_ERR_DIM;
    Bind bind(ctx);
    if (!bind.ok) return WODEN_ERR_CUDA;
    CU(ctx, cudaEventSynchronize(ctx->fit_t1), "fit timing sync");
    CU(ctx, cudaEventElapsedTime(ms, ctx->fit_t0, ctx->fit_t1), "fit timing");
    return WODEN_OK;
}

int woden_shapelet_series(woden_ctx *ctx, int method, int p_max, long long n, const float *x, const float *coeff,
                          double lut_dx, double lut_x_max, float *out, void *cuda_stream)
{
    if (!ctx || !x || !coeff || !out) return WODEN_ERR_NULL;
    if (p_max < 0 || p_max > WODEN_MAX_ORDER) return WODEN_ERR_ORDER;
    if (n <= 0 || (method != WODEN_BASIS_RECURRENCE && method != WODEN_BASIS_LUT)) return WODEN_ERR_DIM;
    Bind bind(ctx);
    if (!bind.ok) return WODEN_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    ctx->last_stream = st;
    int n_x = 0;
    if (method == WODEN_BASIS_LUT) {
        if (!(lut_dx > 0.0) || !(lut_x_max > lut_dx) || lut_x_max / lut_dx > 1 << 22) return WODEN_ERR_DIM;
        n_x = (int)std::ceil(lut_x_max / lut_dx);
        if (ctx->lut_pm != p_max || ctx->lut_nx != n_x || ctx->lut_dx != lut_dx) {       // (re)build the table
            CU(ctx, ctx->lut.reserve((size_t)n_x * (p_max + 1) * sizeof(float2)), "alloc look-up table");
            CU(ctx, launch_lut_build(static_cast<float2 *>(ctx->lut.p), n_x, p_max, lut_dx, st), "table build launch");
            ctx->lut_pm = p_max; ctx->lut_nx = n_x; ctx->lut_dx = lut_dx;
        }
    }
    CU(ctx, launch_series(method, x, coeff, p_max, n, static_cast<const float2 *>(ctx->lut.p), n_x, lut_dx, out, st),
       "series launch");
    return WODEN_OK;
}

int woden_pipe_rate(woden_ctx *ctx, int which, int iters, double *thread_ops_per_s, double *sm_clock_hz)
{
    if (!ctx || !thread_ops_per_s || !sm_clock_hz) return WODEN_ERR_NULL;
    Bind bind(ctx);
    if (!bind.ok) return WODEN_ERR_CUDA;
    CU(ctx, run_pipe_rate(which, iters, thread_ops_per_s, sm_clock_hz), "pipe microbenchmark");
    return WODEN_OK;
}

}  // extern "C"

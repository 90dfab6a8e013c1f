// tm_api.cu -- the C-ABI boundary declared in include/tm.h: handles, validation, dispatch.
// No arithmetic of the method lives here except forming a = 2 kappa mu, b = 2 kappa epsilon and the
// twist coefficients in double (reading C2, C10-ii).
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

#include "tm_internal.h"
#include "tm_layout.cuh"

const TmKernelEntry *tm_generic_table_8_1();
const TmKernelEntry *tm_generic_table_8_2();
const TmKernelEntry *tm_generic_table_4_1();
const TmKernelEntry *tm_generic_table_4_2();
const TmKernelEntry *tm_generic_table_2_1();
const TmKernelEntry *tm_generic_table_2_2();

const TmKernelEntry *tm_tile_table_2_1();
const TmKernelEntry *tm_tile_table_2_2();
const TmKernelEntry *tm_generic_twin_table_8_1();
const TmKernelEntry *tm_generic_twin_table_8_2();
const TmKernelEntry *tm_generic_twin_table_4_1();
const TmKernelEntry *tm_generic_twin_table_4_2();
const TmKernelEntry *tm_generic_twin_table_2_1();
const TmKernelEntry *tm_generic_twin_table_2_2();
const TmKernelEntry *tm_f2_twin_table_4_1();
const TmKernelEntry *tm_f2_twin_table_4_2();
const TmKernelEntry *tm_f2_twin_table_2_1();
const TmKernelEntry *tm_f2_twin_table_2_2();

// input-twist (D R^-1) kernels: packed for fp32 / half unless the scalar path is forced
const TmKernelEntry *tm_twin_table(int prec, int nf, bool packed)
{
    if (prec == 8) return nf == 1 ? tm_generic_twin_table_8_1() : tm_generic_twin_table_8_2();
    if (prec == 4) return packed ? (nf == 1 ? tm_f2_twin_table_4_1() : tm_f2_twin_table_4_2()) : (nf == 1 ? tm_generic_twin_table_4_1() : tm_generic_twin_table_4_2());
    return packed ? (nf == 1 ? tm_f2_twin_table_2_1() : tm_f2_twin_table_2_2()) : (nf == 1 ? tm_generic_twin_table_2_1() : tm_generic_twin_table_2_2());
}

const TmKernelEntry *tm_generic_table(int prec, int nf)
{
    if (prec == 8) return nf == 1 ? tm_generic_table_8_1() : tm_generic_table_8_2();
    if (prec == 4) return nf == 1 ? tm_generic_table_4_1() : tm_generic_table_4_2();
    return nf == 1 ? tm_generic_table_2_1() : tm_generic_table_2_2();
}

const TmKernelEntry *tm_f2_table_4_1();
const TmKernelEntry *tm_f2_table_4_2();
const TmKernelEntry *tm_f2_table_2_1();
const TmKernelEntry *tm_f2_table_2_2();

// packed-FP32 (FFMA2) kernels: fp32 and half only (fp64 has no packed form)
const TmKernelEntry *tm_f2_table(int prec, int nf)
{
    if (prec == 4) return nf == 1 ? tm_f2_table_4_1() : tm_f2_table_4_2();
    if (prec == 2) return nf == 1 ? tm_f2_table_2_1() : tm_f2_table_2_2();
    return nullptr;
}

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

int cuda_fail(cudaError_t e, const char *what)
{
    return fail(TM_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

// Every entry point that allocates, copies or launches selects the context's device first (the caller's current
// device may be another one: two contexts on two GPUs in one thread).
int use_device(const tm_ctx *c)
{
    int cur = -1;
    if (cudaGetDevice(&cur) == cudaSuccess && cur == c->device) return TM_OK;
    cudaError_t e = cudaSetDevice(c->device);
    if (e != cudaSuccess) return cuda_fail(e, "cudaSetDevice");
    return TM_OK;
}
#define TM_USE_DEVICE(c) do { int rc_ = use_device(c); if (rc_) return rc_; } while (0)

bool valid_prec(int p) { return p == TM_DOUBLE || p == TM_SINGLE || p == TM_HALF; }

size_t field_bytes(const TmGeom &g, int prec, int nf)
{
    return (size_t)nf * tm_tiles(g.Vh) * spinor_tile_bytes(prec);      // tiled SoA, the last tile padded (tm_layout.cuh)
}

// The fused D R^-1 kernels (TWIN) replace a separate local pass (read + write of one field) by 8 register twists and full-site
// time hops.  Measured at 32^3 x 64 (profiles/r2_tuning.md section 2), fused against kernel A + local pass: fp64 195 / 189 + 62 us,
// fp32 97 / 95 + 31, half 90 / 78 + 17, fp64 doublet 311 / 273 + 123, fp32 doublet 167 / 150 + 61; only the half doublet, bound by
// the FP32 datapath (176 / 127 + 33), loses and keeps the local pass.
bool fused_twist_in_pays(const tm_field *f) { return !(f->nf == 2 && f->prec == TM_HALF); }

bool overlap(const tm_field *a, const tm_field *b)
{
    const char *pa = static_cast<const char *>(a->ptr), *pb = static_cast<const char *>(b->ptr);
    return pa < pb + b->bytes && pb < pa + a->bytes;
}

// Device staging buffer for upload / download, cached on the context (grown on demand, freed in tm_finalize).
// Safe to reuse: every upload / download synchronises the stream before it returns.
struct Staging {
    tm_ctx *c;
    void *p = nullptr;
    explicit Staging(tm_ctx *ctx) : c(ctx) {}
    cudaError_t alloc(size_t bytes)
    {
        if (c->staging_bytes < bytes) {
            if (c->staging) cudaFree(c->staging);
            c->staging = nullptr;
            c->staging_bytes = 0;
            cudaError_t e = cudaMalloc(&c->staging, bytes);
            if (e != cudaSuccess) return e;
            c->staging_bytes = bytes;
        }
        p = c->staging;
        return cudaSuccess;
    }
};

struct Coeffs {
    double alpha, beta, scale;
};

// a = 2 kappa mu, b = 2 kappa epsilon; R = 1 + i a g5 tau3 + b tau1; R^-1 = (1 - i a g5 tau3 - b tau1)/(1 + a^2 - b^2)
int make_coeffs(const tm_params *p, int nf, int dagger, int kt, Coeffs *c)
{
    if (!(p->t_boundary == 1 || p->t_boundary == -1)) return fail(TM_ERR_PARAM, "t_boundary must be +1 or -1");
    if (nf == 1 && !(p->twist_flavor == 1 || p->twist_flavor == -1))
        return fail(TM_ERR_MISMATCH, "single-flavor fields need twist_flavor = +1 or -1 (got %d)", p->twist_flavor);
    if (nf == 2 && p->twist_flavor != 0)
        return fail(TM_ERR_MISMATCH, "doublet fields need twist_flavor = 0 (got %d)", p->twist_flavor);
    if (nf == 1 && p->epsilon != 0.0) return fail(TM_ERR_PARAM, "epsilon must be 0 for a single flavor (PAPER.md:87)");
    double a = 2.0 * p->kappa * p->mu, b = 2.0 * p->kappa * p->epsilon;
    if (dagger) a = -a;
    if (nf == 1) { a *= (double)p->twist_flavor; b = 0.0; }
    if (kt == TM_DSLASH_XPAY || kt == TM_DSLASH_AXPY || kt == TM_DSLASH_TWIST_INV_AXPY) {       // no (output) twist: the B / REC kernels with R = 1
        c->alpha = 0.0; c->beta = 0.0; c->scale = 1.0;
    } else if (kt == TM_DSLASH_TWIST_XPAY) {
        c->alpha = a; c->beta = b; c->scale = 1.0;
    } else {
        const double den = 1.0 + a * a - b * b;
        if (std::fabs(den) < 1e-12) return fail(TM_ERR_PARAM, "1 + a^2 - b^2 = %g: R is singular", den);
        c->alpha = -a; c->beta = -b; c->scale = 1.0 / den;
    }
    return TM_OK;
}

}  // namespace

extern "C" {

const char *tm_last_error(void) { return g_err; }

int tm_init(const int dims[4], int cuda_device, tm_ctx **ctx)
{
    if (!dims || !ctx) return fail(TM_ERR_ARG, "tm_init: NULL argument");
    *ctx = nullptr;
    for (int d = 0; d < 4; d++)
        if (dims[d] < 4 || (dims[d] & 1)) return fail(TM_ERR_DIMS, "extent %d = %d must be even and >= 4", d, dims[d]);
    const long V = (long)dims[0] * dims[1] * dims[2] * dims[3];
    if (V / 2 > 0x3fffffffL) return fail(TM_ERR_DIMS, "lattice too large for 32-bit site indices");
    cudaError_t e = cudaSetDevice(cuda_device);
    if (e != cudaSuccess) return cuda_fail(e, "cudaSetDevice");
    tm_ctx *c = new (std::nothrow) tm_ctx();
    if (!c) return fail(TM_ERR_NOMEM, "out of host memory");
    for (int d = 0; d < 4; d++) c->g.X[d] = dims[d];
    c->g.Xh = dims[0] / 2;
    c->g.V = V;
    c->g.Vh = (int)(V / 2);
    c->device = cuda_device;
    c->stream = 0;
    c->launches = 0;
    c->last_kernel = "";
    c->path = 0;
    c->pf_dist = -1;
    c->stage = -1;
    c->z_chunks = -1;
    c->tile_kernel = -1;
    c->pdl = 1;
    c->block_threads = 0;
    c->sm_count = 0;
    c->basis_on = 0;
    for (int k = 0; k < 32; k++) c->basis[k] = 0.0;
    c->staging = nullptr;
    c->staging_bytes = 0;
    c->red = nullptr;
    c->red_n = 0;
    c->cgs = nullptr;
    c->cgs_host = nullptr;
    c->cg_ev[0] = c->cg_ev[1] = nullptr;
    c->allreduce = nullptr;
    c->allreduce_user = nullptr;
    c->up_stream = c->down_stream = nullptr;
    c->ev_compute = c->ev_up = c->ev_down = nullptr;
    c->up_staging = c->down_staging = nullptr;
    c->up_bytes = c->down_bytes = 0;
    c->async_ready = false;
    c->open_mask = 0;
    c->halo_counter = nullptr;
    c->timing = false;
    c->timing_chain = false;
    e = cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, cuda_device);
    if (e != cudaSuccess) { delete c; return cuda_fail(e, "cudaDeviceGetAttribute"); }
    *ctx = c;
    return TM_OK;
}

int tm_set_stream(tm_ctx *ctx, void *cuda_stream)
{
    if (!ctx) return fail(TM_ERR_ARG, "tm_set_stream: NULL context");
    ctx->stream = static_cast<cudaStream_t>(cuda_stream);
    return TM_OK;
}

int tm_sync(tm_ctx *ctx)
{
    if (!ctx) return fail(TM_ERR_ARG, "tm_sync: NULL context");
    cudaError_t e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) return cuda_fail(e, "cudaStreamSynchronize");
    if (ctx->async_ready) {        // pending asynchronous uploads / downloads
        if ((e = cudaStreamSynchronize(ctx->up_stream)) != cudaSuccess) return cuda_fail(e, "cudaStreamSynchronize(upload)");
        if ((e = cudaStreamSynchronize(ctx->down_stream)) != cudaSuccess) return cuda_fail(e, "cudaStreamSynchronize(download)");
    }
    return TM_OK;
}

void tm_finalize(tm_ctx *ctx)
{
    if (!ctx) return;
    if (ctx->staging) cudaFree(ctx->staging);
    if (ctx->red) cudaFree(ctx->red);
    if (ctx->async_ready) {
        cudaStreamSynchronize(ctx->up_stream);
        cudaStreamSynchronize(ctx->down_stream);
        cudaStreamDestroy(ctx->up_stream);
        cudaStreamDestroy(ctx->down_stream);
        cudaEventDestroy(ctx->ev_compute);
        cudaEventDestroy(ctx->ev_up);
        cudaEventDestroy(ctx->ev_down);
    }
    if (ctx->up_staging) cudaFree(ctx->up_staging);
    if (ctx->down_staging) cudaFree(ctx->down_staging);
    for (tm_field *f : ctx->cg_ws) tm_field_free(f);
    for (auto e : ctx->cg_ev) if (e) cudaEventDestroy(e);
    if (ctx->cgs) cudaFree(ctx->cgs);
    if (ctx->halo_counter) cudaFree(ctx->halo_counter);
    if (ctx->cgs_host) cudaFreeHost(ctx->cgs_host);
    for (auto &t : ctx->timed) { if (t.own_start) cudaEventDestroy(t.start); cudaEventDestroy(t.stop); }
    delete ctx;
}

static void clear_timed(tm_ctx *ctx)
{
    for (auto &t : ctx->timed) { if (t.own_start) cudaEventDestroy(t.start); cudaEventDestroy(t.stop); }
    ctx->timed.clear();
}

int tm_timing_enable(tm_ctx *ctx, int on)
{
    if (!ctx) return fail(TM_ERR_ARG, "tm_timing_enable: NULL context");
    if (on < 0 || on > 2) return fail(TM_ERR_ARG, "tm_timing_enable: on must be 0, 1 or 2");
    if (on == 0 || (on == 2) != ctx->timing_chain) clear_timed(ctx);
    ctx->timing = on != 0;
    ctx->timing_chain = on == 2;
    return TM_OK;
}

int tm_timing_read(tm_ctx *ctx, int max_records, const char **names, float *ms, int *n)
{
    if (!ctx || !names || !ms || !n || max_records < 0) return fail(TM_ERR_ARG, "tm_timing_read: bad argument");
    cudaError_t e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) return cuda_fail(e, "cudaStreamSynchronize");
    int k = 0;
    for (auto &t : ctx->timed) {
        if (k >= max_records) break;
        float v = 0.f;
        if ((e = cudaEventElapsedTime(&v, t.start, t.stop)) != cudaSuccess) return cuda_fail(e, "cudaEventElapsedTime");
        names[k] = t.name;
        ms[k] = v;
        k++;
    }
    *n = k;
    clear_timed(ctx);
    return TM_OK;
}

int tm_set_host_basis(tm_ctx *ctx, tm_basis basis, const double *custom)
{
    if (!ctx) return fail(TM_ERR_ARG, "tm_set_host_basis: NULL context");
    double m[32];
    for (int k = 0; k < 32; k++) m[k] = 0.0;
    if (basis == TM_BASIS_NONREL) {
        ctx->basis_on = 0;
        return TM_OK;
    } else if (basis == TM_BASIS_CHIRAL) {
        // S = (1 / sqrt 2) [[1, 1], [1, -1]] (2x2 spin blocks): gamma^chiral = S gamma^nonrel S, gamma5^chiral = diag(1,1,-1,-1)
        const double h = 0.70710678118654752440;
        for (int a = 0; a < 2; a++) {
            m[((a) * 4 + a) * 2] = h;
            m[((a) * 4 + a + 2) * 2] = h;
            m[((a + 2) * 4 + a) * 2] = h;
            m[((a + 2) * 4 + a + 2) * 2] = -h;
        }
    } else if (basis == TM_BASIS_CUSTOM) {
        if (!custom) return fail(TM_ERR_ARG, "tm_set_host_basis: TM_BASIS_CUSTOM needs the matrix");
        for (int k = 0; k < 32; k++) m[k] = custom[k];
        for (int a = 0; a < 4; a++)           // S S^dag = 1
            for (int b = 0; b < 4; b++) {
                double re = 0.0, im = 0.0;
                for (int t = 0; t < 4; t++) {
                    const double ar = m[(a * 4 + t) * 2], ai = m[(a * 4 + t) * 2 + 1], br = m[(b * 4 + t) * 2], bi = -m[(b * 4 + t) * 2 + 1];
                    re += ar * br - ai * bi;
                    im += ar * bi + ai * br;
                }
                if (std::fabs(re - (a == b ? 1.0 : 0.0)) > 1e-12 || std::fabs(im) > 1e-12)
                    return fail(TM_ERR_ARG, "tm_set_host_basis: the matrix is not unitary (S S^dag [%d][%d] = %g%+gi)", a, b, re, im);
            }
    } else {
        return fail(TM_ERR_ARG, "tm_set_host_basis: bad basis %d", (int)basis);
    }
    for (int k = 0; k < 32; k++) ctx->basis[k] = m[k];
    ctx->basis_on = 1;
    return TM_OK;
}

int tm_set_path(tm_ctx *ctx, int path)
{
    if (!ctx || path < 0 || path > 1) return fail(TM_ERR_ARG, "tm_set_path: bad argument");
    ctx->path = path;
    return TM_OK;
}

int tm_set_tuning(tm_ctx *ctx, const char *key, int value)
{
    if (!ctx || !key) return fail(TM_ERR_ARG, "tm_set_tuning: NULL argument");
    if (!strcmp(key, "prefetch_blocks")) {
        if (value < -1) return fail(TM_ERR_ARG, "prefetch_blocks must be -1 (default) or >= 0");
        ctx->pf_dist = value;
        return TM_OK;
    }
    if (!strcmp(key, "stage_links")) {
        if (value < -1 || value > 1) return fail(TM_ERR_ARG, "stage_links must be -1 (default), 0 or 1");
        ctx->stage = value;
        return TM_OK;
    }
    if (!strcmp(key, "pdl")) {
        if (value < 0 || value > 1) return fail(TM_ERR_ARG, "pdl must be 0 or 1");
        ctx->pdl = value;
        return TM_OK;
    }
    if (!strcmp(key, "tile_kernel")) {
        if (value < -1 || value > 1) return fail(TM_ERR_ARG, "tile_kernel must be -1 (default), 0 or 1");
        ctx->tile_kernel = value;
        return TM_OK;
    }
    if (!strcmp(key, "z_chunks")) {
        if (value < -1 || value == 0) return fail(TM_ERR_ARG, "z_chunks must be -1 (default) or >= 1");
        ctx->z_chunks = value;
        return TM_OK;
    }
    if (!strcmp(key, "block_threads")) {
        if (value != 0 && value != 32 && value != 64 && value != 128) return fail(TM_ERR_ARG, "block_threads must be 0 (default), 32, 64 or 128");
        ctx->block_threads = value;
        return TM_OK;
    }
    return fail(TM_ERR_ARG, "tm_set_tuning: unknown key '%s'", key);
}

long tm_launch_count(const tm_ctx *ctx) { return ctx ? ctx->launches : 0; }
const char *tm_last_kernel_name(const tm_ctx *ctx) { return ctx ? ctx->last_kernel : ""; }

size_t tm_field_bytes(const tm_ctx *ctx, tm_precision prec, int n_flavor)
{
    if (!ctx || !valid_prec(prec) || n_flavor < 1 || n_flavor > 2) return 0;
    return field_bytes(ctx->g, prec, n_flavor);
}

int tm_field_alloc(tm_ctx *ctx, tm_precision prec, int n_flavor, void *ext_dev_ptr, size_t ext_bytes, tm_field **f)
{
    if (!ctx || !f) return fail(TM_ERR_ARG, "tm_field_alloc: NULL argument");
    *f = nullptr;
    if (!valid_prec(prec)) return fail(TM_ERR_ARG, "bad precision %d", (int)prec);
    if (n_flavor < 1 || n_flavor > 2) return fail(TM_ERR_ARG, "n_flavor must be 1 or 2");
    TM_USE_DEVICE(ctx);
    const size_t bytes = field_bytes(ctx->g, prec, n_flavor);
    tm_field *fl = new (std::nothrow) tm_field();
    if (!fl) return fail(TM_ERR_NOMEM, "out of host memory");
    fl->ctx = ctx; fl->prec = prec; fl->nf = n_flavor; fl->bytes = bytes;
    if (ext_dev_ptr) {
        if (ext_bytes < bytes) { delete fl; return fail(TM_ERR_ARG, "external buffer has %zu bytes, need %zu", ext_bytes, bytes); }
        if (reinterpret_cast<size_t>(ext_dev_ptr) & 255) { delete fl; return fail(TM_ERR_ARG, "external buffer must be 256-byte aligned"); }
        fl->ptr = ext_dev_ptr; fl->owns = false;
    } else {
        cudaError_t e = cudaMalloc(&fl->ptr, bytes);
        if (e != cudaSuccess) { delete fl; cudaGetLastError(); return fail(TM_ERR_NOMEM, "cudaMalloc(%zu): %s", bytes, cudaGetErrorString(e)); }
        fl->owns = true;
    }
    *f = fl;
    return TM_OK;
}

void tm_field_free(tm_field *f)
{
    if (!f) return;
    if (f->owns && f->ptr) cudaFree(f->ptr);
    delete f;
}

void *tm_field_device_ptr(const tm_field *f) { return f ? f->ptr : nullptr; }

static int field_upload(tm_field *f, int parity, const double *host, bool cb)
{
    if (!f || !host) return fail(TM_ERR_ARG, "tm_field_upload: NULL argument");
    if (parity != 0 && parity != 1) return fail(TM_ERR_ARG, "bad parity %d", parity);
    tm_ctx *c = f->ctx;
    TM_USE_DEVICE(c);
    const size_t n = (size_t)f->nf * (cb ? (size_t)c->g.Vh : (size_t)c->g.V) * 24 * sizeof(double);
    Staging st(c);
    cudaError_t e = st.alloc(n);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(TM_ERR_NOMEM, "staging cudaMalloc(%zu): %s", n, cudaGetErrorString(e)); }
    e = cudaMemcpyAsync(st.p, host, n, cudaMemcpyHostToDevice, c->stream);
    if (e != cudaSuccess) return cuda_fail(e, "cudaMemcpyAsync H2D");
    e = tm_pack_spinor(f, parity, st.p, 8, cb, c->stream);
    if (e != cudaSuccess) return cuda_fail(e, "pack_spinor launch");
    e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(e, "upload sync");
    return TM_OK;
}

static int field_download(const tm_field *f, int parity, double *host, bool cb)
{
    if (!f || !host) return fail(TM_ERR_ARG, "tm_field_download: NULL argument");
    if (parity != 0 && parity != 1) return fail(TM_ERR_ARG, "bad parity %d", parity);
    tm_ctx *c = f->ctx;
    TM_USE_DEVICE(c);
    const size_t n = (size_t)f->nf * (cb ? (size_t)c->g.Vh : (size_t)c->g.V) * 24 * sizeof(double);
    Staging st(c);
    cudaError_t e = st.alloc(n);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(TM_ERR_NOMEM, "staging cudaMalloc(%zu): %s", n, cudaGetErrorString(e)); }
    if (!cb) {   // only this parity's sites are written: start from the caller's array
        e = cudaMemcpyAsync(st.p, host, n, cudaMemcpyHostToDevice, c->stream);
        if (e != cudaSuccess) return cuda_fail(e, "cudaMemcpyAsync H2D");
    }
    e = tm_unpack_spinor(f, parity, st.p, 8, cb, c->stream);
    if (e != cudaSuccess) return cuda_fail(e, "unpack_spinor launch");
    e = cudaMemcpyAsync(host, st.p, n, cudaMemcpyDeviceToHost, c->stream);
    if (e != cudaSuccess) return cuda_fail(e, "cudaMemcpyAsync D2H");
    e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(e, "download sync");
    return TM_OK;
}

// ---- asynchronous forms: the copies run on their own streams and overlap the kernels of the context stream and each other ----
static int async_setup(tm_ctx *c)
{
    if (c->async_ready) return TM_OK;
    cudaError_t e;
    if ((e = cudaStreamCreateWithFlags(&c->up_stream, cudaStreamNonBlocking)) != cudaSuccess) return cuda_fail(e, "cudaStreamCreate");
    if ((e = cudaStreamCreateWithFlags(&c->down_stream, cudaStreamNonBlocking)) != cudaSuccess) return cuda_fail(e, "cudaStreamCreate");
    for (cudaEvent_t *ev : {&c->ev_compute, &c->ev_up, &c->ev_down})
        if ((e = cudaEventCreateWithFlags(ev, cudaEventDisableTiming)) != cudaSuccess) return cuda_fail(e, "cudaEventCreate");
    c->async_ready = true;
    return TM_OK;
}

static cudaError_t grow(void **p, size_t *have, size_t need, cudaStream_t owner)
{
    if (*have >= need) return cudaSuccess;
    cudaError_t e = cudaStreamSynchronize(owner);        // the old buffer may still be in use by queued copies
    if (e != cudaSuccess) return e;
    if (*p) cudaFree(*p);
    *p = nullptr;
    *have = 0;
    e = cudaMalloc(p, need);
    if (e == cudaSuccess) *have = need;
    return e;
}

static int upload_cb_async(tm_field *f, tm_parity parity, const void *host_cb, int host_prec)
{
    if (!f || !host_cb) return fail(TM_ERR_ARG, "tm_field_upload_cb_async: NULL argument");
    if (parity != TM_EVEN && parity != TM_ODD) return fail(TM_ERR_ARG, "bad parity %d", (int)parity);
    tm_ctx *c = f->ctx;
    TM_USE_DEVICE(c);
    int rc = async_setup(c);
    if (rc) return rc;
    const size_t n = (size_t)f->nf * (size_t)c->g.Vh * 24 * (size_t)host_prec;
    cudaError_t e = grow(&c->up_staging, &c->up_bytes, n, c->up_stream);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(TM_ERR_NOMEM, "staging cudaMalloc(%zu): %s", n, cudaGetErrorString(e)); }
    // H2D copy: free to run now (the staging buffer is ordered by the upload stream itself)
    if ((e = cudaMemcpyAsync(c->up_staging, host_cb, n, cudaMemcpyHostToDevice, c->up_stream)) != cudaSuccess) return cuda_fail(e, "cudaMemcpyAsync H2D");
    // the pack kernel overwrites f: it waits for every kernel already queued on the context stream (they may read f)
    if ((e = cudaEventRecord(c->ev_compute, c->stream)) != cudaSuccess) return cuda_fail(e, "cudaEventRecord");
    if ((e = cudaStreamWaitEvent(c->up_stream, c->ev_compute, 0)) != cudaSuccess) return cuda_fail(e, "cudaStreamWaitEvent");
    if ((e = tm_pack_spinor(f, (int)parity, c->up_staging, host_prec, true, c->up_stream)) != cudaSuccess) return cuda_fail(e, "pack_spinor launch");
    // later kernels of the context stream see the uploaded field
    if ((e = cudaEventRecord(c->ev_up, c->up_stream)) != cudaSuccess) return cuda_fail(e, "cudaEventRecord");
    if ((e = cudaStreamWaitEvent(c->stream, c->ev_up, 0)) != cudaSuccess) return cuda_fail(e, "cudaStreamWaitEvent");
    return TM_OK;
}

static int download_cb_async(const tm_field *f, tm_parity parity, void *host_cb, int host_prec)
{
    if (!f || !host_cb) return fail(TM_ERR_ARG, "tm_field_download_cb_async: NULL argument");
    if (parity != TM_EVEN && parity != TM_ODD) return fail(TM_ERR_ARG, "bad parity %d", (int)parity);
    tm_ctx *c = f->ctx;
    TM_USE_DEVICE(c);
    int rc = async_setup(c);
    if (rc) return rc;
    const size_t n = (size_t)f->nf * (size_t)c->g.Vh * 24 * (size_t)host_prec;
    cudaError_t e = grow(&c->down_staging, &c->down_bytes, n, c->down_stream);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(TM_ERR_NOMEM, "staging cudaMalloc(%zu): %s", n, cudaGetErrorString(e)); }
    // the unpack kernel reads f after everything queued on the context stream so far
    if ((e = cudaEventRecord(c->ev_compute, c->stream)) != cudaSuccess) return cuda_fail(e, "cudaEventRecord");
    if ((e = cudaStreamWaitEvent(c->down_stream, c->ev_compute, 0)) != cudaSuccess) return cuda_fail(e, "cudaStreamWaitEvent");
    if ((e = tm_unpack_spinor(f, (int)parity, c->down_staging, host_prec, true, c->down_stream)) != cudaSuccess) return cuda_fail(e, "unpack_spinor launch");
    // later kernels of the context stream may overwrite f once it has been unpacked; the D2H copy itself overlaps them
    if ((e = cudaEventRecord(c->ev_down, c->down_stream)) != cudaSuccess) return cuda_fail(e, "cudaEventRecord");
    if ((e = cudaStreamWaitEvent(c->stream, c->ev_down, 0)) != cudaSuccess) return cuda_fail(e, "cudaStreamWaitEvent");
    if ((e = cudaMemcpyAsync(host_cb, c->down_staging, n, cudaMemcpyDeviceToHost, c->down_stream)) != cudaSuccess) return cuda_fail(e, "cudaMemcpyAsync D2H");
    return TM_OK;
}

int tm_field_upload_cb_async(tm_field *f, tm_parity parity, const double *host_cb) { return upload_cb_async(f, parity, host_cb, 8); }
int tm_field_download_cb_async(const tm_field *f, tm_parity parity, double *host_cb) { return download_cb_async(f, parity, host_cb, 8); }
int tm_field_upload_cb_async_f32(tm_field *f, tm_parity parity, const float *host_cb) { return upload_cb_async(f, parity, host_cb, 4); }
int tm_field_download_cb_async_f32(const tm_field *f, tm_parity parity, float *host_cb) { return download_cb_async(f, parity, host_cb, 4); }

int tm_field_upload(tm_field *f, tm_parity parity, const double *host_full) { return field_upload(f, parity, host_full, false); }
int tm_field_download(const tm_field *f, tm_parity parity, double *host_full) { return field_download(f, parity, host_full, false); }
int tm_field_upload_cb(tm_field *f, tm_parity parity, const double *host_cb) { return field_upload(f, parity, host_cb, true); }
int tm_field_download_cb(const tm_field *f, tm_parity parity, double *host_cb) { return field_download(f, parity, host_cb, true); }

int tm_gauge_load(tm_ctx *ctx, const double *host_links, tm_precision prec, tm_recon recon, tm_gauge **g)
{
    if (!ctx || !host_links || !g) return fail(TM_ERR_ARG, "tm_gauge_load: NULL argument");
    *g = nullptr;
    if (!valid_prec(prec)) return fail(TM_ERR_ARG, "bad precision %d", (int)prec);
    if (recon != TM_RECON_18 && recon != TM_RECON_12 && recon != TM_RECON_8) return fail(TM_ERR_ARG, "bad recon %d", (int)recon);
    if (recon == TM_RECON_8) {
        // The 8-real chart divides by N = |U01|^2 + |U02|^2 (tm_layout.cuh: rebuild_from8): a rounding / storage error eps of the
        // stored reals comes back as eps / N in the rebuilt row 1.  eps: 1e-16 (fp64), ~5e-7 (fp32: the packed kernels rebuild with
        // the fast sin / cos / rcp units), 3e-5 (half: int16 storage).  The bound keeps the worst single link's error below
        // 1e-8 / 5e-2 / 3 (x its magnitude): links closer to the chart's singular point are refused, not silently degraded
        // further.  (Haar links: P(N < d) = d^2, so 32^3 x 64 has ~0.3 links below 1e-4 and none below 1e-5 in expectation.)
        const double nmin_ok = (int)prec == TM_DOUBLE ? 1e-8 : 1e-5;
        const size_t nl = (size_t)4 * ctx->g.V;
        double nmin = 1.0;
        for (size_t l = 0; l < nl; l++) {
            const double *u = host_links + l * 18;
            const double N = u[2] * u[2] + u[3] * u[3] + u[4] * u[4] + u[5] * u[5];
            if (N < nmin) nmin = N;
        }
        if (!(nmin >= nmin_ok))
            return fail(TM_ERR_PARAM, "8-real links: a link has |U01|^2 + |U02|^2 = %.3g < %.0e, too close to the chart's singular point for "
                                      "this precision (use 12- or 18-real)", nmin, nmin_ok);
    }
    TM_USE_DEVICE(ctx);
    tm_gauge *gg = new (std::nothrow) tm_gauge();
    if (!gg) return fail(TM_ERR_NOMEM, "out of host memory");
    gg->ctx = ctx; gg->prec = prec; gg->recon = recon;
    gg->bytes = (size_t)2 * tm_tiles(ctx->g.Vh) * 4 * link_tile_bytes(prec, recon);
    cudaError_t e = cudaMalloc(&gg->ptr, gg->bytes);
    if (e != cudaSuccess) { delete gg; cudaGetLastError(); return fail(TM_ERR_NOMEM, "cudaMalloc(%zu): %s", gg->bytes, cudaGetErrorString(e)); }
    const size_t n = (size_t)4 * ctx->g.V * 18 * sizeof(double);
    Staging st(ctx);
    e = st.alloc(n);
    if (e != cudaSuccess) { tm_gauge_free(gg); cudaGetLastError(); return fail(TM_ERR_NOMEM, "staging cudaMalloc(%zu): %s", n, cudaGetErrorString(e)); }
    e = cudaMemcpyAsync(st.p, host_links, n, cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = tm_pack_gauge(gg, static_cast<const double *>(st.p), ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) { tm_gauge_free(gg); return cuda_fail(e, "tm_gauge_load"); }
    *g = gg;
    return TM_OK;
}

void tm_gauge_free(tm_gauge *g)
{
    if (!g) return;
    if (g->ptr) cudaFree(g->ptr);
    delete g;
}

int tm_dslash_apply(tm_field *out, const tm_field *in, const tm_field *x, const tm_gauge *g, const tm_params *p,
                    tm_parity parity, int dagger, tm_kernel_type kt, tm_precision prec)
{
    if (!out || !in || !g || !p) return fail(TM_ERR_ARG, "tm_dslash_apply: NULL argument");
    if (parity != TM_EVEN && parity != TM_ODD) return fail(TM_ERR_ARG, "bad parity %d", (int)parity);
    if ((int)kt < 0 || (int)kt > 8) return fail(TM_ERR_ARG, "bad kernel type %d", (int)kt);
    // out = x - kappa^2 D in  and  out = x + kappa D in  run the B / REC kernels with the identity twist; the D R^-1 forms
    // (kt 6, 7, 8) run the A / REC kernels with the inverse twist applied to the input sites (TWIN)
    const bool twin = (int)kt >= (int)TM_TWIST_INV_DSLASH_TWIST_INV;
    const int kcode = kt == TM_DSLASH_XPAY ? (int)TM_DSLASH_TWIST_XPAY : (kt == TM_DSLASH_AXPY || kt == TM_RECONSTRUCT_TWIST_INV || kt == TM_DSLASH_TWIST_INV_AXPY) ? (int)TM_RECONSTRUCT
                      : kt == TM_TWIST_INV_DSLASH_TWIST_INV ? (int)TM_TWIST_INV_DSLASH : (int)kt;
    if (kt != TM_TWIST_INV_DSLASH && kt != TM_TWIST_INV_DSLASH_TWIST_INV && !x) return fail(TM_ERR_ARG, "kernel type %d needs x", (int)kt);
    tm_ctx *c = out->ctx;
    if (in->ctx != c || g->ctx != c || (x && x->ctx != c)) return fail(TM_ERR_MISMATCH, "operands belong to different contexts");
    if (out->prec != (int)prec || in->prec != (int)prec || g->prec != (int)prec || (x && x->prec != (int)prec))
        return fail(TM_ERR_MISMATCH, "precision mismatch (call %d, out %d, in %d, gauge %d)", (int)prec, out->prec, in->prec, g->prec);
    if (in->nf != out->nf || (x && x->nf != out->nf)) return fail(TM_ERR_MISMATCH, "flavor count mismatch");
    if (overlap(out, in)) return fail(TM_ERR_ALIAS, "out aliases in");
    if (x && overlap(out, x) && out->ptr != x->ptr) return fail(TM_ERR_ALIAS, "out partially overlaps x (only out == x is allowed)");
    TM_USE_DEVICE(c);
    Coeffs co;
    int rc = make_coeffs(p, out->nf, dagger ? 1 : 0, (int)kt, &co);
    if (rc) return rc;

    DslashArgs a;
    a.out = out->ptr; a.in = in->ptr; a.x = x ? x->ptr : nullptr; a.gauge = g->ptr;
    a.X = c->g.X[0]; a.Y = c->g.X[1]; a.Z = c->g.X[2]; a.T = c->g.X[3]; a.Xh = c->g.Xh; a.Vh = c->g.Vh;
    a.dXh = tm_fastdiv(a.Xh); a.dY = tm_fastdiv(a.Y); a.dZ = tm_fastdiv(a.Z);
    a.parity = (int)parity;
    a.alpha = co.alpha; a.beta = co.beta; a.scale = co.scale;
    a.alpha_in = 0.0; a.beta_in = 0.0; a.scale_in = 1.0;
    if (twin) {
        Coeffs ci;
        rc = make_coeffs(p, out->nf, dagger ? 1 : 0, (int)TM_TWIST_INV_DSLASH, &ci);       // R^-1 (R^dag^-1 when daggered) on the input
        if (rc) return rc;
        a.alpha_in = ci.alpha; a.beta_in = ci.beta; a.scale_in = ci.scale;
    }
    a.kappa = p->kappa; a.kappa2 = p->kappa * p->kappa;
    a.tbound = (c->open_mask & 8) ? 0.0 : (double)p->t_boundary;      // cut directions: the wrapped hops come from tm_halo_apply
    a.wrap_y = (c->open_mask & 2) ? 0.f : 1.f;
    a.wrap_z = (c->open_mask & 4) ? 0.f : 1.f;
    // measured defaults (profiles/): the fp64 doublet kernels with 12-real links gain from an L2 prefetch 8 tiles ahead, the half
    // kernels from staging the link stream through shared memory; everything else runs plain
    // L2 prefetch of the tiles 8 blocks ahead (tm_stream.cuh), where it measured faster at both 32^3 x 64 and 48^3 x 96 (profiles/r2_tuning.md
    // section 5): the fp32 doublet kernels (+6..11 %), the fp64 kernels without an x input (+2..5 %), the fp64 doublet with 12-real links
    const bool pf_on = ((int)prec == TM_SINGLE && out->nf == 2) || ((int)prec == TM_DOUBLE && (kcode == 0 || (out->nf == 2 && g->recon == 12)));
    a.pdl = c->pdl;
    a.pf_dist = c->pf_dist >= 0 ? c->pf_dist : (pf_on ? 8 : 0);
    int stage = c->stage >= 0 ? c->stage : ((int)prec == TM_HALF ? 1 : 0);
    a.block_threads = c->block_threads ? c->block_threads : 128;
    if (g->recon == 8 || twin) stage = 0;        // 8-real links and the D R^-1 kernels: direct loads
    while (stage && (size_t)8 * g->recon * (int)prec * a.block_threads > 96 * 1024 && a.block_threads > 32) a.block_threads /= 2;

    // z-chunked traversal: the input spinor is re-read over a window of three time slices; when those (next to the streaming
    // links and the output) do not fit the L2, the lattice is walked in chunks of Z / nzc z-planes (profiles/r2_tuning.md)
    {
        const size_t slice = (size_t)c->g.Xh * c->g.X[1] * c->g.X[2];                          // sites of one parity per time slice
        const size_t window = 3 * slice * (size_t)out->nf * 24 * (int)prec;
        int nzc = c->z_chunks >= 1 ? c->z_chunks : 1;
        if (c->z_chunks < 0)
            while (window / nzc > (size_t)40 << 20 && nzc < c->g.X[2]) nzc *= 2;
        while (nzc > 1 && (c->g.X[2] % nzc != 0 || (slice / nzc) % a.block_threads != 0 || slice / nzc / a.block_threads < 2)) nzc--;
        a.nzc = nzc;
        a.bpz = (int)(slice / nzc / a.block_threads);
        if (nzc > 1) { a.dbpc = tm_fastdiv(a.bpz * c->g.X[3]); a.dbpz = tm_fastdiv(a.bpz); }
        else { a.dbpc = tm_fastdiv(2); a.dbpz = tm_fastdiv(2); }
    }

    // path 0: fp32 / half run the packed-FP32 kernels, fp64 the scalar kernel; path 1 forces the scalar kernel
    // (8-real links: packed kernels with direct loads only)
    const int kidx = (((g->recon == 18 ? 0 : g->recon == 12 ? 1 : 2) * 4 + kcode) * 2 + (dagger ? 1 : 0)) * 2 + stage;
    const TmKernelEntry *tab = (c->path == 0 && (int)prec != TM_DOUBLE) ? tm_f2_table((int)prec, out->nf) : nullptr;
    if (!tab || !tab[kidx].fn) tab = tm_generic_table((int)prec, out->nf);
    // half precision: the warp-per-tile kernel with shared-memory staged operands (tm_dslash_tile.cuh) where the lattice allows it.
    // Measured (profiles/r2_tuning.md section 4): 6-7 % faster than the staged thread-per-site kernel for one flavor, 2-4 % for the doublet
    // (26 KB of shared memory per warp, 8 warps per SM): the default wherever the geometry fits ("tile_kernel" = 0 turns it off)
    const bool tile = (int)prec == TM_HALF && c->path == 0 && !twin && g->recon != 8 && c->tile_kernel != 0 &&
                      (c->g.Xh == 4 || c->g.Xh == 8 || c->g.Xh == 16) && c->g.X[1] % (32 / c->g.Xh) == 0 && c->g.Vh % 32 == 0;
    const TmKernelEntry &k = tile ? (out->nf == 1 ? tm_tile_table_2_1() : tm_tile_table_2_2())[((g->recon == 18 ? 0 : 1) * 4 + kcode) * 2 + (dagger ? 1 : 0)]
                           : twin ? tm_twin_table((int)prec, out->nf, c->path == 0)[((g->recon == 18 ? 0 : g->recon == 12 ? 1 : 2) * 2 + (kcode == 3 ? 1 : 0)) * 2 + (dagger ? 1 : 0)]
                                  : tab[kidx];
    cudaError_t e;
    if (c->timing) {
        tm_ctx::TimedLaunch t;
        t.name = k.name;
        t.own_start = !(c->timing_chain && !c->timed.empty());
        if (t.own_start) {
            if ((e = cudaEventCreate(&t.start)) != cudaSuccess) return cuda_fail(e, "cudaEventCreate");
        } else {
            t.start = c->timed.back().stop;            // chained: the event between the previous launch and this one
        }
        if ((e = cudaEventCreate(&t.stop)) != cudaSuccess) { if (t.own_start) cudaEventDestroy(t.start); return cuda_fail(e, "cudaEventCreate"); }
        if (t.own_start) cudaEventRecord(t.start, c->stream);
        e = k.fn(a, c->stream);
        cudaEventRecord(t.stop, c->stream);
        c->timed.push_back(t);
    } else {
        e = k.fn(a, c->stream);
    }
    if (e != cudaSuccess) return cuda_fail(e, k.name);
    c->launches++;
    c->last_kernel = k.name;
    return TM_OK;
}

int tm_mat_pc(tm_field *out_e, const tm_field *in_e, tm_field *tmp_o, const tm_gauge *g, const tm_params *p,
              tm_matpc type, int dagger)
{
    if (!out_e || !in_e || !tmp_o || !g || !p) return fail(TM_ERR_ARG, "tm_mat_pc: NULL argument");
    if (type != TM_MATPC_ASYM && type != TM_MATPC_SYM) return fail(TM_ERR_ARG, "bad matpc type %d", (int)type);
    if (overlap(tmp_o, in_e) || overlap(tmp_o, out_e)) return fail(TM_ERR_ALIAS, "tmp_o aliases in_e or out_e");
    const tm_precision prec = (tm_precision)out_e->prec;
    if (type == TM_MATPC_SYM && dagger) {
        // M^_sym^dag = 1 - kappa^2 D^dag_eo R^dag^-1_oo D^dag_oe R^dag^-1_ee  (C7): the twist stands in FRONT of the first
        // hopping term: the fused D R^-1 kernel applies it to the neighbour sites in registers.
        if (overlap(out_e, in_e)) return fail(TM_ERR_ALIAS, "out_e aliases in_e");
        int rc;
        if (fused_twist_in_pays(out_e)) {
            rc = tm_dslash_apply(tmp_o, in_e, nullptr, g, p, TM_ODD, 1, TM_TWIST_INV_DSLASH_TWIST_INV, prec);   // tmp_o = R^dag^-1 D^dag R^dag^-1 in_e
        } else {
            rc = tm_twist_apply(out_e, in_e, p, 1, 1);                                                           // out_e = R^dag^-1 in_e (scratch)
            if (!rc) rc = tm_dslash_apply(tmp_o, out_e, nullptr, g, p, TM_ODD, 1, TM_TWIST_INV_DSLASH, prec);
        }
        if (!rc) rc = tm_dslash_apply(out_e, tmp_o, in_e, g, p, TM_EVEN, 1, TM_DSLASH_XPAY, prec);               // out_e = in_e - kappa^2 D^dag tmp_o
        return rc;
    }
    // tmp_o = R_oo^-1 D_oe in_e
    int rc = tm_dslash_apply(tmp_o, in_e, nullptr, g, p, TM_ODD, dagger, TM_TWIST_INV_DSLASH, prec);
    if (rc) return rc;
    // ASYM: out_e = R_ee in_e - kappa^2 D_eo tmp_o ;  SYM: out_e = in_e - kappa^2 R_ee^-1 D_eo tmp_o
    return tm_dslash_apply(out_e, tmp_o, in_e, g, p, TM_EVEN, dagger,
                           type == TM_MATPC_ASYM ? TM_DSLASH_TWIST_XPAY : TM_TWIST_INV_DSLASH_XPAY, prec);
}

int tm_twist_apply(tm_field *out, const tm_field *in, const tm_params *p, int inverse, int dagger)
{
    if (!out || !in || !p) return fail(TM_ERR_ARG, "tm_twist_apply: NULL argument");
    tm_ctx *c = out->ctx;
    if (in->ctx != c) return fail(TM_ERR_MISMATCH, "operands belong to different contexts");
    if (in->prec != out->prec || in->nf != out->nf) return fail(TM_ERR_MISMATCH, "precision or flavor count mismatch");
    if (overlap(out, in) && out->ptr != in->ptr) return fail(TM_ERR_ALIAS, "out partially overlaps in");
    TM_USE_DEVICE(c);
    Coeffs co;
    int rc = make_coeffs(p, out->nf, dagger ? 1 : 0, inverse ? (int)TM_TWIST_INV_DSLASH : (int)TM_DSLASH_TWIST_XPAY, &co);
    if (rc) return rc;
    cudaError_t e = tm_launch_twist(out, in, co.alpha, co.beta, co.scale, c->stream);
    if (e != cudaSuccess) return cuda_fail(e, "tm_twist_kernel");
    c->launches++;
    c->last_kernel = "twist";
    return TM_OK;
}

int tm_prepare_rhs(tm_field *rhs_e, const tm_field *b_e, const tm_field *b_o, tm_field *tmp_o, const tm_gauge *g,
                   const tm_params *p, tm_matpc type)
{
    if (!rhs_e || !b_e || !b_o || !tmp_o || !g || !p) return fail(TM_ERR_ARG, "tm_prepare_rhs: NULL argument");
    if (type != TM_MATPC_ASYM && type != TM_MATPC_SYM) return fail(TM_ERR_ARG, "bad matpc type %d", (int)type);
    if (overlap(tmp_o, b_e) || overlap(tmp_o, rhs_e) || overlap(tmp_o, b_o)) return fail(TM_ERR_ALIAS, "tmp_o aliases b_e, b_o or rhs_e");
    const tm_precision prec = (tm_precision)rhs_e->prec;
    // Eq. 2.2: b_e + kappa D_eo R_oo^-1 b_o ;  Eq. 2.3: R_ee^-1 (b_e + kappa D_eo R_oo^-1 b_o)   (reading C4)
    if (!fused_twist_in_pays(rhs_e)) {
        int rc = tm_twist_apply(tmp_o, b_o, p, 1, 0);                                     // tmp_o = R_oo^-1 b_o
        if (rc) return rc;
        return tm_dslash_apply(rhs_e, tmp_o, b_e, g, p, TM_EVEN, 0, type == TM_MATPC_ASYM ? TM_DSLASH_AXPY : TM_RECONSTRUCT, prec);
    }
    // one launch of the fused D R^-1 kernel; tmp_o is not needed
    return tm_dslash_apply(rhs_e, b_o, b_e, g, p, TM_EVEN, 0, type == TM_MATPC_ASYM ? TM_DSLASH_TWIST_INV_AXPY : TM_RECONSTRUCT_TWIST_INV, prec);
}

// ---- domain decomposition in y, z, t ---------------------------------------------------------
int tm_set_open_dirs(tm_ctx *ctx, int mask)
{
    if (!ctx) return fail(TM_ERR_ARG, "tm_set_open_dirs: NULL context");
    if (mask & ~14) return fail(TM_ERR_ARG, "tm_set_open_dirs: mask %d has bits other than 2 (y), 4 (z), 8 (t)", mask);
    ctx->open_mask = mask;
    return TM_OK;
}

int tm_set_open_time(tm_ctx *ctx, int on) { return tm_set_open_dirs(ctx, on ? 8 : 0); }

size_t tm_halo_bytes(const tm_ctx *ctx, tm_precision prec, int n_flavor, int dir)
{
    if (!ctx || !valid_prec(prec) || (n_flavor != 1 && n_flavor != 2) || dir < 1 || dir > 3) return 0;
    return (size_t)n_flavor * (size_t)(ctx->g.Vh / ctx->g.X[dir]) * 12 * ((int)prec == TM_DOUBLE ? sizeof(double) : sizeof(float));
}

int tm_halo_pack(const tm_field *in, const tm_gauge *g, tm_parity out_parity, int dagger, int dir, void *dev_to_prev, void *dev_to_next,
                 unsigned *dev_flag_prev, unsigned *dev_flag_next, unsigned epoch)
{
    if (!in || !g || !dev_to_prev || !dev_to_next) return fail(TM_ERR_ARG, "tm_halo_pack: NULL argument");
    if (out_parity != TM_EVEN && out_parity != TM_ODD) return fail(TM_ERR_ARG, "bad parity %d", (int)out_parity);
    if (dir < 1 || dir > 3) return fail(TM_ERR_ARG, "tm_halo_pack: dir %d is not 1 (y), 2 (z) or 3 (t)", dir);
    tm_ctx *c = in->ctx;
    if (g->ctx != c) return fail(TM_ERR_MISMATCH, "operands belong to different contexts");
    if (g->prec != in->prec) return fail(TM_ERR_MISMATCH, "precision mismatch (field %d, gauge %d)", in->prec, g->prec);
    TM_USE_DEVICE(c);
    if ((dev_flag_prev || dev_flag_next) && !c->halo_counter) {
        cudaError_t e = cudaMalloc(&c->halo_counter, sizeof(unsigned));
        if (e == cudaSuccess) e = cudaMemsetAsync(c->halo_counter, 0, sizeof(unsigned), c->stream);
        if (e != cudaSuccess) return cuda_fail(e, "halo counter");
    }
    cudaError_t e = tm_launch_halo_pack(in, g, (int)out_parity, dagger ? 1 : 0, dir, dev_to_prev, dev_to_next, dev_flag_prev, dev_flag_next,
                                        epoch, c->halo_counter, c->stream);
    if (e != cudaSuccess) return cuda_fail(e, "halo_pack launch");
    c->launches++;
    c->last_kernel = "halo_pack";
    return TM_OK;
}

int tm_halo_apply(tm_field *out, const void *dev_from_prev, const void *dev_from_next, const tm_gauge *g, const tm_params *p,
                  tm_parity out_parity, int dagger, tm_kernel_type kt, int dir, int sign_prev, int sign_next,
                  const unsigned *dev_wait_prev, const unsigned *dev_wait_next, unsigned epoch)
{
    if (!out || !dev_from_prev || !dev_from_next || !g || !p) return fail(TM_ERR_ARG, "tm_halo_apply: NULL argument");
    if (out_parity != TM_EVEN && out_parity != TM_ODD) return fail(TM_ERR_ARG, "bad parity %d", (int)out_parity);
    if ((int)kt < 0 || (int)kt > 5) return fail(TM_ERR_ARG, "bad kernel type %d (the D R^-1 forms have no distributed completion)", (int)kt);
    if (dir < 1 || dir > 3) return fail(TM_ERR_ARG, "tm_halo_apply: dir %d is not 1 (y), 2 (z) or 3 (t)", dir);
    if ((sign_prev != 1 && sign_prev != -1) || (sign_next != 1 && sign_next != -1)) return fail(TM_ERR_ARG, "boundary signs must be +1 or -1");
    if (dir != 3 && (sign_prev != 1 || sign_next != 1)) return fail(TM_ERR_ARG, "space is periodic: boundary signs must be +1 for dir %d", dir);
    tm_ctx *c = out->ctx;
    if (g->ctx != c) return fail(TM_ERR_MISMATCH, "operands belong to different contexts");
    if (g->prec != out->prec) return fail(TM_ERR_MISMATCH, "precision mismatch (field %d, gauge %d)", out->prec, g->prec);
    TM_USE_DEVICE(c);
    Coeffs co;
    int rc = make_coeffs(p, out->nf, dagger ? 1 : 0, (int)kt, &co);
    if (rc) return rc;
    // the epilogues are affine in the hopping sum (tm_dslash.cuh: epilogue): A: twist(acc); A-xpay: -kappa^2 twist(acc);
    // B and XPAY: -kappa^2 acc; REC and AXPY: twist(kappa acc)
    const int kcode = kt == TM_DSLASH_XPAY ? (int)TM_DSLASH_TWIST_XPAY : kt == TM_DSLASH_AXPY ? (int)TM_RECONSTRUCT : (int)kt;
    const double k2 = p->kappa * p->kappa;
    const double coef = kcode == 0 ? 1.0 : kcode == 3 ? p->kappa : -k2;
    const double hopw = dir == 3 ? 2.0 : 1.0;                      // (1 -+ gamma_4) keeps half the spinor with weight 2
    cudaError_t e = tm_launch_halo_apply(out, dev_from_prev, dev_from_next, g, (int)out_parity, dagger ? 1 : 0, dir, hopw * sign_prev,
                                         hopw * sign_next, co.alpha, co.beta, co.scale, coef, kcode != 2, dev_wait_prev, dev_wait_next,
                                         epoch, c->stream);
    if (e != cudaSuccess) return cuda_fail(e, "halo_apply launch");
    c->launches++;
    c->last_kernel = "halo_apply";
    return TM_OK;
}

int tm_reconstruct_odd(tm_field *psi_o, const tm_field *psi_e, const tm_field *b_o, const tm_gauge *g, const tm_params *p)
{
    if (!psi_o || !psi_e || !b_o || !g || !p) return fail(TM_ERR_ARG, "tm_reconstruct_odd: NULL argument");
    return tm_dslash_apply(psi_o, psi_e, b_o, g, p, TM_ODD, 0, TM_RECONSTRUCT, (tm_precision)psi_o->prec);
}

// ---- vector operations and the mixed-precision CG --------------------

int tm_field_axpby(tm_field *z, double a, const tm_field *x, double b, const tm_field *y)
{
    if (!z || !x) return fail(TM_ERR_ARG, "tm_field_axpby: NULL argument");
    if (x->ctx != z->ctx || (y && y->ctx != z->ctx)) return fail(TM_ERR_MISMATCH, "operands belong to different contexts");
    if (x->nf != z->nf || (y && y->nf != z->nf)) return fail(TM_ERR_MISMATCH, "flavor count mismatch");
    if ((overlap(z, x) && z->ptr != x->ptr) || (y && overlap(z, y) && z->ptr != y->ptr))
        return fail(TM_ERR_ALIAS, "z partially overlaps an input");
    cudaError_t e = tm_blas_axpbyz(z, a, x, b, y, nullptr);
    if (e == cudaErrorInvalidValue) return fail(TM_ERR_UNSUPPORTED, "precision mix (z %d, x %d, y %d) not supported", z->prec, x->prec, y ? y->prec : 0);
    if (e != cudaSuccess) return cuda_fail(e, "tm_field_axpby");
    return TM_OK;
}

int tm_field_redot(const tm_field *x, const tm_field *y, double *result)
{
    if (!x || !y || !result) return fail(TM_ERR_ARG, "tm_field_redot: NULL argument");
    if (x->ctx != y->ctx) return fail(TM_ERR_MISMATCH, "operands belong to different contexts");
    if (x->nf != y->nf || x->prec != y->prec) return fail(TM_ERR_MISMATCH, "precision or flavor count mismatch");
    cudaError_t e = tm_blas_redot(x, y, result);
    if (e != cudaSuccess) return cuda_fail(e, "tm_field_redot");
    return TM_OK;
}

int tm_field_redot_noalloc(const tm_field *x, const tm_field *y, double *dev_result)
{
    if (!x || !y || !dev_result) return fail(TM_ERR_ARG, "tm_field_redot_noalloc: NULL argument");
    if (x->ctx != y->ctx) return fail(TM_ERR_MISMATCH, "operands belong to different contexts");
    if (x->nf != y->nf || x->prec != y->prec) return fail(TM_ERR_MISMATCH, "precision or flavor count mismatch");
    if ((long)x->ctx->g.Vh > TM_NOALLOC_MAX_SITES)
        return fail(TM_ERR_UNSUPPORTED, "tm_field_redot_noalloc: %d sites per parity exceed the fixed scratch array's maximum of %ld "
                                        "(TM_NOALLOC_MAX_SITES); use tm_field_redot", x->ctx->g.Vh, TM_NOALLOC_MAX_SITES);
    cudaError_t e = tm_noalloc_redot(x, y, dev_result);
    if (e != cudaSuccess) return cuda_fail(e, "tm_field_redot_noalloc");
    return TM_OK;
}

namespace {

// Work fields of tm_invert_cg: library-owned device memory kept on the context between solves (zero-filled once so that tile
// padding is defined).  Slot k of a (precision, flavors) pair is created on first use.
tm_field *ws_field(tm_ctx *c, int prec, int nf, int k)
{
    int seen = 0;
    for (tm_field *f : c->cg_ws)
        if (f->prec == prec && f->nf == nf && seen++ == k) return f;
    tm_field *p = nullptr;
    if (tm_field_alloc(c, (tm_precision)prec, nf, nullptr, 0, &p) != TM_OK) return nullptr;
    if (cudaMemsetAsync(p->ptr, 0, p->bytes, c->stream) != cudaSuccess) { tm_field_free(p); return nullptr; }
    c->cg_ws.push_back(p);
    return p;
}

#define TM_TRY_CUDA(call, what) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, what); } while (0)
#define TM_TRY(call) do { int rc_ = (call); if (rc_) return rc_; } while (0)

// out = M^dag M in on the even sites; t_e and tmp_o are scratch of in's precision
int apply_normal(tm_field *out, const tm_field *in, tm_field *t_e, tm_field *tmp_o, const tm_gauge *g, const tm_params *p, tm_matpc type,
                 const tm_cg_params *cp)
{
    if (cp->op) {
        if (cp->op(t_e, in, tmp_o, g, p, type, 0, cp->op_user)) return fail(TM_ERR_CUDA, "tm_invert_cg: the caller's operator failed");
        if (cp->op(out, t_e, tmp_o, g, p, type, 1, cp->op_user)) return fail(TM_ERR_CUDA, "tm_invert_cg: the caller's operator failed");
        return TM_OK;
    }
    int rc = tm_mat_pc(t_e, in, tmp_o, g, p, type, 0);
    if (!rc) rc = tm_mat_pc(out, t_e, tmp_o, g, p, type, 1);
    return rc;
}

}  // namespace

int tm_set_allreduce(tm_ctx *ctx, tm_allreduce_fn fn, void *user)
{
    if (!ctx) return fail(TM_ERR_ARG, "tm_set_allreduce: NULL context");
    ctx->allreduce = fn;
    ctx->allreduce_user = user;
    return TM_OK;
}

void tm_cg_release(tm_ctx *ctx)
{
    if (!ctx) return;
    cudaStreamSynchronize(ctx->stream);
    for (tm_field *f : ctx->cg_ws) tm_field_free(f);
    ctx->cg_ws.clear();
}

int tm_invert_cg(tm_field *x_e, const tm_field *b_e, const tm_gauge *g_precise, const tm_gauge *g_sloppy, const tm_params *p,
                 tm_matpc type, const tm_cg_params *cp, tm_cg_info *info)
{
    if (!x_e || !b_e || !g_precise || !p || !cp || !info) return fail(TM_ERR_ARG, "tm_invert_cg: NULL argument");
    info->iterations = 0; info->restarts = 0; info->residual = 0.0; info->converged = 0;
    tm_ctx *c = x_e->ctx;
    if (b_e->ctx != c || g_precise->ctx != c) return fail(TM_ERR_MISMATCH, "operands belong to different contexts");
    if (x_e->prec != TM_DOUBLE || b_e->prec != TM_DOUBLE || g_precise->prec != TM_DOUBLE)
        return fail(TM_ERR_MISMATCH, "x_e, b_e and g_precise must be double precision");
    if (x_e->nf != b_e->nf) return fail(TM_ERR_MISMATCH, "flavor count mismatch");
    if (overlap(x_e, b_e)) return fail(TM_ERR_ALIAS, "x_e aliases b_e");
    const int ps = (int)cp->sloppy_precision;
    if (!valid_prec(ps)) return fail(TM_ERR_ARG, "bad sloppy precision %d", ps);
    const tm_gauge *gs = ps == TM_DOUBLE ? g_precise : g_sloppy;
    if (!gs || gs->ctx != c || gs->prec != ps) return fail(TM_ERR_MISMATCH, "g_sloppy must be a gauge handle of the sloppy precision");
    if (!(cp->tol > 0.0) || cp->max_iter < 1 || !(cp->delta > 0.0 && cp->delta < 1.0))
        return fail(TM_ERR_ARG, "need tol > 0, max_iter >= 1, 0 < delta < 1");
    if (type != TM_MATPC_ASYM && type != TM_MATPC_SYM) return fail(TM_ERR_ARG, "bad matpc type %d", (int)type);
    const int nf = x_e->nf;
    TM_USE_DEVICE(c);

    // double: residual, A x, two scratch fields; sloppy: residual, direction, A p, partial solution, two scratch fields
    const int d0 = ps == TM_DOUBLE ? 4 : 0;        // sloppy = double: the two sets share one pool
    tm_field *r_d = ws_field(c, TM_DOUBLE, nf, 0), *t_d = ws_field(c, TM_DOUBLE, nf, 1), *te_d = ws_field(c, TM_DOUBLE, nf, 2), *to_d = ws_field(c, TM_DOUBLE, nf, 3);
    tm_field *r_s = ws_field(c, ps, nf, d0 + 0), *p_s = ws_field(c, ps, nf, d0 + 1), *ap_s = ws_field(c, ps, nf, d0 + 2), *x_s = ws_field(c, ps, nf, d0 + 3);
    tm_field *te_s = ps == TM_DOUBLE ? te_d : ws_field(c, ps, nf, 4), *to_s = ps == TM_DOUBLE ? to_d : ws_field(c, ps, nf, 5);
    if (!r_d || !t_d || !te_d || !to_d || !r_s || !p_s || !ap_s || !x_s || !te_s || !to_s) return fail(TM_ERR_NOMEM, "tm_invert_cg: work fields");

    if (!c->cgs) TM_TRY_CUDA(cudaMalloc(&c->cgs, 4 * sizeof(double)), "cudaMalloc(cg scalars)");
    if (!c->cgs_host) TM_TRY_CUDA(cudaHostAlloc(&c->cgs_host, 6 * sizeof(double), cudaHostAllocDefault), "cudaHostAlloc(cg scalars)");
    if (!c->cg_ev[0])
        for (auto &e : c->cg_ev) TM_TRY_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming), "cudaEventCreate");

    double bnorm2 = 0.0, rnorm2 = 0.0;
    TM_TRY_CUDA(tm_blas_redot(b_e, b_e, &bnorm2), "redot");
    TM_TRY_CUDA(tm_blas_axpbyz(x_e, 0.0, b_e, 0.0, nullptr, nullptr), "zero x");        // x = 0
    if (bnorm2 == 0.0) { info->converged = 1; return TM_OK; }
    TM_TRY_CUDA(tm_blas_axpbyz(r_d, 1.0, b_e, 0.0, nullptr, nullptr), "copy b");          // r = b
    rnorm2 = bnorm2;

    // One CG recurrence in the sloppy precision with DEVICE-RESIDENT scalars: alpha = |r|^2 / <p, A p> and beta = |r_new|^2 / |r|^2
    // are formed inside the update kernels from c->cgs, so no step waits for the host.  The scalars of every iteration are copied
    // to a pinned ring and the host looks at them ONE ITERATION LATE (by then they have arrived): the reliable-update decision,
    // the stopping test and the breakdown test lag by one iteration.
    double *sc = c->cgs, *hs = c->cgs_host;
    TM_TRY_CUDA(tm_blas_axpbyz(r_s, 1.0, r_d, 0.0, nullptr, nullptr), "r_s = r");
    TM_TRY_CUDA(tm_blas_axpbyz(p_s, 1.0, r_s, 0.0, nullptr, nullptr), "p = r_s");
    TM_TRY_CUDA(tm_blas_axpbyz(x_s, 0.0, r_s, 0.0, nullptr, nullptr), "x_s = 0");
    int cur = 0;
    TM_TRY_CUDA(tm_blas_redot_dev(r_s, r_s, nullptr, sc + cur), "|r_s|^2");
    double rmax = std::sqrt(rnorm2), last_true = rnorm2;
    int stagnant = 0, update = 0, stop = 0;
    auto look = [&](int slot, int rr_idx) -> int {                        // the scalars of an iteration whose copy has landed
        TM_TRY_CUDA(cudaEventSynchronize(c->cg_ev[slot]), "cg scalars");
        const double pap = hs[3 * slot + 2], rr_new = hs[3 * slot + rr_idx];
        if (!(pap > 0.0)) return fail(TM_ERR_PARAM, "tm_invert_cg: <p, A p> = %g is not positive (breakdown)", pap);
        if (!(rr_new >= 0.0)) return fail(TM_ERR_PARAM, "tm_invert_cg: |r|^2 = %g (breakdown)", rr_new);
        const double rn = std::sqrt(rr_new);
        if (rn < cp->delta * rmax || rn <= cp->tol * std::sqrt(bnorm2)) update = 1;
        if (rn > rmax) rmax = rn;
        return TM_OK;
    };
    int prev_idx = 0;
    for (int it = 0;; it++) {
        TM_TRY(apply_normal(ap_s, p_s, te_s, to_s, gs, p, type, cp));                                                  // A p
        TM_TRY_CUDA(tm_blas_redot_dev(p_s, ap_s, nullptr, sc + 2), "redot");                                             // <p, A p>
        TM_TRY_CUDA(tm_blas_cg_update_dev(x_s, r_s, p_s, ap_s, 0.0, nullptr, sc + cur, sc + 2, sc + (1 - cur)), "cg_update");
        TM_TRY_CUDA(cudaMemcpyAsync(hs + 3 * (it & 1), sc, 3 * sizeof(double), cudaMemcpyDeviceToHost, c->stream), "cg scalars");
        TM_TRY_CUDA(cudaEventRecord(c->cg_ev[it & 1], c->stream), "cg scalars");
        info->iterations++;
        if (it > 0) TM_TRY(look((it - 1) & 1, prev_idx));
        prev_idx = 1 - cur;
        const bool last = info->iterations >= cp->max_iter;
        if (last) TM_TRY(look(it & 1, prev_idx));                           // the final iteration's scalars (breakdown test)
        if (update || last) {
            // reliable update: x += x_s, x_s = 0, r = b - A x in double replaces the iterated residual; the direction is kept
            TM_TRY_CUDA(tm_blas_axpbyz(x_e, 1.0, x_s, 1.0, x_e, nullptr), "x += x_s");
            TM_TRY_CUDA(tm_blas_axpbyz(x_s, 0.0, r_s, 0.0, nullptr, nullptr), "x_s = 0");
            TM_TRY(apply_normal(t_d, x_e, te_d, to_d, g_precise, p, type, cp));
            TM_TRY_CUDA(tm_blas_axpbyz(r_d, 1.0, b_e, -1.0, t_d, &rnorm2), "r = b - A x");
            info->restarts++;
            info->residual = std::sqrt(rnorm2 / bnorm2);
            if (info->residual <= cp->tol) { info->converged = 1; stop = 1; }
            stagnant = rnorm2 > 0.81 * last_true ? stagnant + 1 : 0;       // the true residual must keep falling (by 10 % at least)
            if (stagnant >= 3) stop = 1;                                  // e.g. a half-precision recurrence below its own noise
            last_true = rnorm2;
            if (stop || last) break;
            TM_TRY_CUDA(tm_blas_axpbyz(r_s, 1.0, r_d, 0.0, nullptr, nullptr), "r_s = r");
            TM_TRY_CUDA(tm_blas_redot_dev(r_s, r_s, nullptr, sc + (1 - cur)), "|r_s|^2");
            rmax = std::sqrt(rnorm2);
            update = 0;
        }
        TM_TRY_CUDA(tm_blas_axpbyz_dev(p_s, 1.0, r_s, 0.0, p_s, nullptr, sc + (1 - cur), sc + cur), "xpay");            // p = r_s + beta p
        cur = 1 - cur;
    }
    return TM_OK;
}

}  // extern "C"

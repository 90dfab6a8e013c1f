// tm_blas.cu -- the vector operations of the mixed-precision CG ("mixed precision CG inverter")
// on single-parity fields in the tiled layout: z = a x + b y (any mix of precisions, optional |z|^2), Re<x, y>, and
// the fused CG update  x += a p, r -= a Ap, |r|^2.  One thread per site (every flavor of the site); reductions are
// deterministic: per-block partial sums in double, then one block adds them in a fixed order.
// Half fields are dequantised with their site norms on load and requantised on store (tm_layout.cuh).
#include "tm_internal.h"
#include "tm_layout.cuh"

namespace {

constexpr int BT = 128;          // threads per block

// block sum of one double per thread -> partial[blockIdx.x] (thread 0)
__device__ __forceinline__ void block_sum(double v, double *partial)
{
    __shared__ double sh[BT / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0;
#pragma unroll
        for (int w = 0; w < BT / 32; w++) s += sh[w];
        partial[blockIdx.x] = s;
    }
}

// out[0] = sum of partial[0..n) in index order (one block; each thread takes a strided slice, then a fixed tree)
__global__ void __launch_bounds__(256) final_sum_kernel(const double *partial, int n, double *out)
{
    __shared__ double sh[256];
    double s = 0;
    for (int i = threadIdx.x; i < n; i += 256) s += partial[i];
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[0] = sh[0];
}

template <int PZ, int PX, int PY, int NF, bool NORM>
__global__ void __launch_bounds__(BT) axpbyz_kernel(char *z, double a, const char *x, double b, const char *y, int Vh, double *partial,
                                                    const double *bnum, const double *bden)
{
    if (bnum) b = *bnum / *bden;                 // device-resident scalar (inner CG: beta = |r_new|^2 / |r|^2)
    const int site = blockIdx.x * BT + threadIdx.x;
    double n2 = 0;
    if (site < Vh) {
        const int lane = site & (TM_TILE - 1);
#pragma unroll
        for (int f = 0; f < NF; f++) {
            typename PrecTraits<PX>::real vx[24];
            double w[24];
            load_spinor<PX, 0>(vx, x + spinor_site_off(PX, NF, site, f), lane);
#pragma unroll
            for (int i = 0; i < 24; i++) w[i] = a * (double)vx[i];
            if (y) {
                typename PrecTraits<PY>::real vy[24];
                load_spinor<PY, 0>(vy, y + spinor_site_off(PY, NF, site, f), lane);
#pragma unroll
                for (int i = 0; i < 24; i++) w[i] += b * (double)vy[i];
            }
            typename PrecTraits<PZ>::real vz[24];
#pragma unroll
            for (int i = 0; i < 24; i++) {
                vz[i] = (typename PrecTraits<PZ>::real)w[i];
                if (NORM) n2 += w[i] * w[i];
            }
            store_spinor<PZ>(vz, z + spinor_site_off(PZ, NF, site, f), lane);
        }
    }
    if (NORM) block_sum(n2, partial);
}

template <int P, int NF>
__global__ void __launch_bounds__(BT) redot_kernel(const char *x, const char *y, int Vh, double *partial)
{
    const int site = blockIdx.x * BT + threadIdx.x;
    double s = 0;
    if (site < Vh) {
        const int lane = site & (TM_TILE - 1);
#pragma unroll
        for (int f = 0; f < NF; f++) {
            typename PrecTraits<P>::real vx[24], vy[24];
            load_spinor<P, 0>(vx, x + spinor_site_off(P, NF, site, f), lane);
            load_spinor<P, 0>(vy, y + spinor_site_off(P, NF, site, f), lane);
#pragma unroll
            for (int i = 0; i < 24; i++) s += (double)vx[i] * (double)vy[i];
        }
    }
    block_sum(s, partial);
}

// x += a p ; r -= a Ap ; partial |r|^2
template <int P, int NF>
__global__ void __launch_bounds__(BT) cg_update_kernel(char *x, char *r, const char *p, const char *Ap, double a, int Vh, double *partial,
                                                       const double *anum, const double *aden)
{
    typedef typename PrecTraits<P>::real real;
    if (anum) a = *anum / *aden;                 // device-resident scalar (inner CG: alpha = |r|^2 / <p, A p>)
    const int site = blockIdx.x * BT + threadIdx.x;
    double n2 = 0;
    if (site < Vh) {
        const int lane = site & (TM_TILE - 1);
#pragma unroll
        for (int f = 0; f < NF; f++) {
            const size_t off = spinor_site_off(P, NF, site, f);
            real vx[24], vr[24], vp[24], va[24];
            load_spinor<P, 0>(vx, x + off, lane);
            load_spinor<P, 0>(vp, p + off, lane);
            load_spinor<P, 0>(vr, r + off, lane);
            load_spinor<P, 0>(va, Ap + off, lane);
#pragma unroll
            for (int i = 0; i < 24; i++) {
                vx[i] = (real)((double)vx[i] + a * (double)vp[i]);
                const double t = (double)vr[i] - a * (double)va[i];
                vr[i] = (real)t;
                n2 += t * t;
            }
            store_spinor<P>(vx, x + off, lane);
            store_spinor<P>(vr, r + off, lane);
        }
    }
    block_sum(n2, partial);
}

cudaError_t reduce_buffers(tm_ctx *c, int blocks)
{
    if (c->red_n < (size_t)blocks + 1) {
        if (c->red) cudaFree(c->red);
        c->red = nullptr;
        c->red_n = 0;
        cudaError_t e = cudaMalloc(&c->red, ((size_t)blocks + 1) * sizeof(double));
        if (e != cudaSuccess) return e;
        c->red_n = (size_t)blocks + 1;
    }
    return cudaSuccess;
}

// multi-GPU: the caller's all-reduce (tm_set_allreduce) sums the device word over the ranks, in stream order
cudaError_t global_sum(tm_ctx *c, double *dev_word)
{
    if (!c->allreduce) return cudaSuccess;
    return c->allreduce(dev_word, 1, static_cast<void *>(c->stream), c->allreduce_user) == 0 ? cudaSuccess : cudaErrorUnknown;
}

// partials are in c->red[1..blocks]; the sum goes to *dev_out and stays on the device (no synchronisation)
cudaError_t finish_sum_dev(tm_ctx *c, int blocks, double *dev_out)
{
    final_sum_kernel<<<1, 256, 0, c->stream>>>(c->red + 1, blocks, dev_out);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    return global_sum(c, dev_out);
}

// partials are in c->red[1..blocks]; the sum goes to c->red[0] and from there to *host (synchronises the stream)
cudaError_t finish_sum(tm_ctx *c, int blocks, double *host)
{
    final_sum_kernel<<<1, 256, 0, c->stream>>>(c->red + 1, blocks, c->red);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if ((e = global_sum(c, c->red)) != cudaSuccess) return e;
    e = cudaMemcpyAsync(host, c->red, sizeof(double), cudaMemcpyDeviceToHost, c->stream);
    if (e != cudaSuccess) return e;
    return cudaStreamSynchronize(c->stream);
}

}  // namespace

// z = a x + b y (y may be NULL: z = a x); operands may have different precisions but the same flavor count.
// Supported mixes: all equal; z double with x sloppy and y double; z sloppy with x double (y NULL or of z's precision).
cudaError_t tm_blas_axpbyz(tm_field *z, double a, const tm_field *x, double b, const tm_field *y, double *norm2)
{
    return tm_blas_axpbyz_dev(z, a, x, b, y, norm2, nullptr, nullptr);
}

// the same with b = *bnum / *bden read on the device when bnum != NULL (DEVICE pointers)
cudaError_t tm_blas_axpbyz_dev(tm_field *z, double a, const tm_field *x, double b, const tm_field *y, double *norm2,
                               const double *bnum, const double *bden)
{
    tm_ctx *c = z->ctx;
    const int Vh = c->g.Vh, blocks = (Vh + BT - 1) / BT;
    cudaError_t e = reduce_buffers(c, blocks);
    if (e != cudaSuccess) return e;
    char *zp = static_cast<char *>(z->ptr);
    const char *xp = static_cast<const char *>(x->ptr), *yp = y ? static_cast<const char *>(y->ptr) : nullptr;
    const int pz = z->prec, px = x->prec, py = y ? y->prec : pz;
    bool done = false;
#define TM_AX(PZ, PX, PY)                                                                                             \
    if (!done && pz == PZ && px == PX && py == PY) {                                                                  \
        done = true;                                                                                                  \
        if (z->nf == 1) { if (norm2) axpbyz_kernel<PZ, PX, PY, 1, true><<<blocks, BT, 0, c->stream>>>(zp, a, xp, b, yp, Vh, c->red + 1, bnum, bden);   \
                          else axpbyz_kernel<PZ, PX, PY, 1, false><<<blocks, BT, 0, c->stream>>>(zp, a, xp, b, yp, Vh, c->red + 1, bnum, bden); }     \
        else            { if (norm2) axpbyz_kernel<PZ, PX, PY, 2, true><<<blocks, BT, 0, c->stream>>>(zp, a, xp, b, yp, Vh, c->red + 1, bnum, bden);   \
                          else axpbyz_kernel<PZ, PX, PY, 2, false><<<blocks, BT, 0, c->stream>>>(zp, a, xp, b, yp, Vh, c->red + 1, bnum, bden); }     \
    }
    TM_AX(8, 8, 8) TM_AX(4, 4, 4) TM_AX(2, 2, 2)
    TM_AX(8, 4, 8) TM_AX(8, 2, 8)            // x_double += a * e_sloppy
    TM_AX(4, 8, 4) TM_AX(2, 8, 2)            // r_sloppy = a * r_double
#undef TM_AX
    if (!done) return cudaErrorInvalidValue;
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    c->launches++;
    c->last_kernel = "blas_axpbyz";
    return norm2 ? finish_sum(c, blocks, norm2) : cudaSuccess;
}

cudaError_t tm_blas_redot(const tm_field *x, const tm_field *y, double *out) { return tm_blas_redot_dev(x, y, out, nullptr); }

// dev_out != NULL: the sum is left in *dev_out (DEVICE pointer), nothing is copied back and the stream is not synchronised
cudaError_t tm_blas_redot_dev(const tm_field *x, const tm_field *y, double *out, double *dev_out)
{
    tm_ctx *c = x->ctx;
    const int Vh = c->g.Vh, blocks = (Vh + BT - 1) / BT;
    cudaError_t e = reduce_buffers(c, blocks);
    if (e != cudaSuccess) return e;
    const char *xp = static_cast<const char *>(x->ptr), *yp = static_cast<const char *>(y->ptr);
#define TM_DOT(P, N) redot_kernel<P, N><<<blocks, BT, 0, c->stream>>>(xp, yp, Vh, c->red + 1)
    if (x->prec == 8) { if (x->nf == 1) TM_DOT(8, 1); else TM_DOT(8, 2); }
    else if (x->prec == 4) { if (x->nf == 1) TM_DOT(4, 1); else TM_DOT(4, 2); }
    else { if (x->nf == 1) TM_DOT(2, 1); else TM_DOT(2, 2); }
#undef TM_DOT
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    c->launches++;
    c->last_kernel = "blas_redot";
    return dev_out ? finish_sum_dev(c, blocks, dev_out) : finish_sum(c, blocks, out);
}

cudaError_t tm_blas_cg_update(tm_field *x, tm_field *r, const tm_field *p, const tm_field *Ap, double a, double *rr)
{
    return tm_blas_cg_update_dev(x, r, p, Ap, a, rr, nullptr, nullptr, nullptr);
}

// anum != NULL: a = *anum / *aden on the device and |r|^2 is left in *dev_rr (DEVICE pointers), no synchronisation
cudaError_t tm_blas_cg_update_dev(tm_field *x, tm_field *r, const tm_field *p, const tm_field *Ap, double a, double *rr,
                                  const double *anum, const double *aden, double *dev_rr)
{
    tm_ctx *c = x->ctx;
    const int Vh = c->g.Vh, blocks = (Vh + BT - 1) / BT;
    cudaError_t e = reduce_buffers(c, blocks);
    if (e != cudaSuccess) return e;
    char *xp = static_cast<char *>(x->ptr), *rp = static_cast<char *>(r->ptr);
    const char *pp = static_cast<const char *>(p->ptr), *ap = static_cast<const char *>(Ap->ptr);
#define TM_UP(P, N) cg_update_kernel<P, N><<<blocks, BT, 0, c->stream>>>(xp, rp, pp, ap, a, Vh, c->red + 1, anum, aden)
    if (x->prec == 8) { if (x->nf == 1) TM_UP(8, 1); else TM_UP(8, 2); }
    else if (x->prec == 4) { if (x->nf == 1) TM_UP(4, 1); else TM_UP(4, 2); }
    else { if (x->nf == 1) TM_UP(2, 1); else TM_UP(2, 2); }
#undef TM_UP
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    c->launches++;
    c->last_kernel = "blas_cg_update";
    return dev_rr ? finish_sum_dev(c, blocks, dev_rr) : finish_sum(c, blocks, rr);
}

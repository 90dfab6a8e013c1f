// tm_pack.cu -- host canonical order (double) <-> device checkerboard SoA (row a1 of DESIGN.md).
// Not on the hot path: runs once per upload / download.  Sources are device staging copies of the host arrays.
#include "tm_internal.h"
#include "tm_layout.cuh"

namespace {

struct PackGeom {
    int X, Y, Z, T, Xh, Vh;
    long V;
};

// host spin basis (tm_set_host_basis): w = S v (ADJ = false) or S^dag v (ADJ = true) on the spin index, color by color
struct SpinRot {
    int on;
    double m[32];        // S[row][col][re, im]
};
template <bool ADJ>
__device__ __forceinline__ void spin_rotate(double *v, const SpinRot &r)
{
    double w[24];
#pragma unroll
    for (int s = 0; s < 4; s++)
#pragma unroll
        for (int c = 0; c < 3; c++) {
            double re = 0.0, im = 0.0;
#pragma unroll
            for (int t = 0; t < 4; t++) {
                const double mr = ADJ ? r.m[(t * 4 + s) * 2] : r.m[(s * 4 + t) * 2];
                const double mi = ADJ ? -r.m[(t * 4 + s) * 2 + 1] : r.m[(s * 4 + t) * 2 + 1];
                const double xr = v[(t * 3 + c) * 2], xi = v[(t * 3 + c) * 2 + 1];
                re += mr * xr - mi * xi;
                im += mr * xi + mi * xr;
            }
            w[(s * 3 + c) * 2] = re;
            w[(s * 3 + c) * 2 + 1] = im;
        }
#pragma unroll
    for (int k = 0; k < 24; k++) v[k] = w[k];
}

__device__ __forceinline__ long cb_to_lex(const PackGeom &g, int i, int parity)
{
    int r = i / g.Xh;
    const int y = r % g.Y;
    r /= g.Y;
    const int z = r % g.Z;
    const int t = r / g.Z;
    return 2L * i + ((y + z + t + parity) & 1);      // lex / 2 == i, x1 parity fixed by the row
}

// HT = the host array's real type: double (the canonical form) or float (tm_field_upload_cb_async_f32: half the PCIe bytes)
template <int PREC, typename HT>
__global__ void pack_spinor_kernel(char *dst, const HT *src, PackGeom g, int parity, int nf, bool src_is_cb, SpinRot rot)
{
    typedef typename PrecTraits<PREC>::real real;
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= nf * g.Vh) return;
    const int f = tid / g.Vh, i = tid % g.Vh;
    const HT *s = src_is_cb ? src + ((size_t)f * g.Vh + i) * 24 : src + ((size_t)f * g.V + cb_to_lex(g, i, parity)) * 24;
    double d[24];
#pragma unroll
    for (int k = 0; k < 24; k++) d[k] = (double)s[k];
    if (rot.on) spin_rotate<false>(d, rot);
    real v[24];
#pragma unroll
    for (int k = 0; k < 24; k++) v[k] = (real)d[k];
    store_spinor<PREC>(v, dst + spinor_site_off(PREC, nf, i, f), i & (TM_TILE - 1));
}

template <int PREC, typename HT>
__global__ void unpack_spinor_kernel(HT *dst, const char *src, PackGeom g, int parity, int nf, bool dst_is_cb, SpinRot rot)
{
    typedef typename PrecTraits<PREC>::real real;
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= nf * g.Vh) return;
    const int f = tid / g.Vh, i = tid % g.Vh;
    real v[24];
    load_spinor<PREC, 0>(v, src + spinor_site_off(PREC, nf, i, f), i & (TM_TILE - 1));
    HT *d = dst_is_cb ? dst + ((size_t)f * g.Vh + i) * 24 : dst + ((size_t)f * g.V + cb_to_lex(g, i, parity)) * 24;
    double o[24];
#pragma unroll
    for (int k = 0; k < 24; k++) o[k] = (double)v[k];
    if (rot.on) spin_rotate<true>(o, rot);
#pragma unroll
    for (int k = 0; k < 24; k++) d[k] = (HT)o[k];
}

// one thread per (parity, mu, cb site): U_mu(x) for x of that parity
template <int PREC, int RECON>
__global__ void pack_gauge_kernel(char *dst, const double *src, PackGeom g)
{
    const long tid = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 8L * g.Vh) return;
    const int i = (int)(tid % g.Vh);
    const int pm = (int)(tid / g.Vh);       // parity * 4 + mu
    const int parity = pm >> 2, mu = pm & 3;
    const double *s = src + ((size_t)mu * g.V + cb_to_lex(g, i, parity)) * 18;
    char *lp = dst + (size_t)parity * tm_tiles(g.Vh) * 4 * link_tile_bytes(PREC, RECON) + link_site_off(PREC, RECON, i, mu);
    const int lane = i & (TM_TILE - 1);
    if constexpr (RECON == 8) {
        // the chart of rebuild_from8 (tm_layout.cuh): a2, a3, b1, arg(a1) / pi, arg(c1) / pi
        const double p[8] = {s[2], s[3], s[4], s[5], s[6], s[7], atan2(s[1], s[0]) / M_PI, atan2(s[13], s[12]) / M_PI};
        if constexpr (PREC == 8) {
#pragma unroll
            for (int k = 0; k < 4; k++) *reinterpret_cast<double2 *>(lp + k * TM_PLANE) = make_double2(p[2 * k], p[2 * k + 1]);
        } else if constexpr (PREC == 4) {
#pragma unroll
            for (int k = 0; k < 2; k++)
                *reinterpret_cast<float4 *>(lp + k * TM_PLANE) =
                    make_float4((float)p[4 * k], (float)p[4 * k + 1], (float)p[4 * k + 2], (float)p[4 * k + 3]);
        } else {
            int w[4];
#pragma unroll
            for (int k = 0; k < 4; k++) w[k] = pack2((float)p[2 * k] * TM_HALF_MAX, (float)p[2 * k + 1] * TM_HALF_MAX);
            *reinterpret_cast<int4 *>(lp) = make_int4(w[0], w[1], w[2], w[3]);
        }
    } else if constexpr (PREC == 8) {
#pragma unroll
        for (int k = 0; k < RECON / 2; k++)
            *reinterpret_cast<double2 *>(lp + k * TM_PLANE) = make_double2(s[2 * k], s[2 * k + 1]);
    } else if constexpr (PREC == 4) {
        constexpr int NF4 = (RECON == 18) ? 4 : 3;
#pragma unroll
        for (int k = 0; k < NF4; k++)
            *reinterpret_cast<float4 *>(lp + k * TM_PLANE) =
                make_float4((float)s[4 * k], (float)s[4 * k + 1], (float)s[4 * k + 2], (float)s[4 * k + 3]);
        if constexpr (RECON == 18)
            *reinterpret_cast<float2 *>(lp + tail_off(4, 8, lane)) = make_float2((float)s[16], (float)s[17]);
    } else {
        int w[9];
#pragma unroll
        for (int k = 0; k < RECON / 2; k++)
            w[k] = pack2((float)s[2 * k] * TM_HALF_MAX, (float)s[2 * k + 1] * TM_HALF_MAX);
        *reinterpret_cast<int4 *>(lp) = make_int4(w[0], w[1], w[2], w[3]);
        if constexpr (RECON == 18) {
            *reinterpret_cast<int4 *>(lp + TM_PLANE) = make_int4(w[4], w[5], w[6], w[7]);
            *reinterpret_cast<int *>(lp + tail_off(2, 4, lane)) = w[8];
        } else {
            *reinterpret_cast<int2 *>(lp + tail_off(1, 8, lane)) = make_int2(w[4], w[5]);
        }
    }
}

SpinRot rot_of(const tm_ctx *c)
{
    SpinRot r;
    r.on = c->basis_on;
    for (int k = 0; k < 32; k++) r.m[k] = c->basis[k];
    return r;
}

PackGeom geom_of(const tm_ctx *c)
{
    PackGeom g;
    g.X = c->g.X[0];
    g.Y = c->g.X[1];
    g.Z = c->g.X[2];
    g.T = c->g.X[3];
    g.Xh = c->g.Xh;
    g.Vh = c->g.Vh;
    g.V = c->g.V;
    return g;
}

}  // namespace

cudaError_t tm_pack_spinor(const tm_field *f, int parity, const void *dev_src, int host_prec, bool src_is_cb, cudaStream_t s)
{
    const PackGeom g = geom_of(f->ctx);
    const SpinRot rot = rot_of(f->ctx);
    const int n = f->nf * g.Vh, threads = 128, blocks = (n + threads - 1) / threads;
    char *dst = static_cast<char *>(f->ptr);
#define TM_PS(P, HT) pack_spinor_kernel<P, HT><<<blocks, threads, 0, s>>>(dst, static_cast<const HT *>(dev_src), g, parity, f->nf, src_is_cb, rot)
    if (host_prec == 8) { if (f->prec == 8) TM_PS(8, double); else if (f->prec == 4) TM_PS(4, double); else TM_PS(2, double); }
    else { if (f->prec == 8) TM_PS(8, float); else if (f->prec == 4) TM_PS(4, float); else TM_PS(2, float); }
#undef TM_PS
    return cudaGetLastError();
}

cudaError_t tm_unpack_spinor(const tm_field *f, int parity, void *dev_dst, int host_prec, bool dst_is_cb, cudaStream_t s)
{
    const PackGeom g = geom_of(f->ctx);
    const SpinRot rot = rot_of(f->ctx);
    const int n = f->nf * g.Vh, threads = 128, blocks = (n + threads - 1) / threads;
    const char *src = static_cast<const char *>(f->ptr);
#define TM_US(P, HT) unpack_spinor_kernel<P, HT><<<blocks, threads, 0, s>>>(static_cast<HT *>(dev_dst), src, g, parity, f->nf, dst_is_cb, rot)
    if (host_prec == 8) { if (f->prec == 8) TM_US(8, double); else if (f->prec == 4) TM_US(4, double); else TM_US(2, double); }
    else { if (f->prec == 8) TM_US(8, float); else if (f->prec == 4) TM_US(4, float); else TM_US(2, float); }
#undef TM_US
    return cudaGetLastError();
}

cudaError_t tm_pack_gauge(const tm_gauge *gg, const double *dev_src, cudaStream_t s)
{
    const PackGeom g = geom_of(gg->ctx);
    const long n = 8L * g.Vh;
    const int threads = 128, blocks = (int)((n + threads - 1) / threads);
    char *dst = static_cast<char *>(gg->ptr);
#define TM_PG(P, R) pack_gauge_kernel<P, R><<<blocks, threads, 0, s>>>(dst, dev_src, g)
    if (gg->prec == 8) { if (gg->recon == 18) TM_PG(8, 18); else if (gg->recon == 12) TM_PG(8, 12); else TM_PG(8, 8); }
    else if (gg->prec == 4) { if (gg->recon == 18) TM_PG(4, 18); else if (gg->recon == 12) TM_PG(4, 12); else TM_PG(4, 8); }
    else { if (gg->recon == 18) TM_PG(2, 18); else if (gg->recon == 12) TM_PG(2, 12); else TM_PG(2, 8); }
#undef TM_PG
    return cudaGetLastError();
}

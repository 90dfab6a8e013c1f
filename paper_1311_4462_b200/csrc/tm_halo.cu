// tm_halo.cu -- time-direction domain decomposition ("packing routines for the
// communication buffers", :134 multi-GPU runs): the lattice is cut into slabs along x4, one slab per GPU.  The fused dslash
// kernels run on the slab with the time hops that leave it switched off (tm_set_open_time); this file supplies the two
// surface kernels around the exchange:
//   halo_pack  : spin-projected half-spinors (12 reals per site and flavor -- the doublet's face carries the flavor index)
//                of the first time slice (for the previous slab's forward hops) and U_4^dag times the half-spinors of the
//                last time slice (for the next slab's backward hops: the link lives with the sender)
//   halo_apply : adds the missing hops to the boundary sites of the kernel's output.  Every fused epilogue is affine in the
//                hopping sum, so out += coef * [twist](acc_surface) completes A, A-xpay, B, REC and the twist-free forms.
// Face site j of a time slice = checkerboard index inside the slice; the site at x4 = T-1 and its +t neighbour in the next
// slab have the same j (tm_dslash.cuh: tp = site - (T-1) * st), so sender and receiver index the buffers identically.
// Buffers hold double (fp64 fields) or float (fp32 and half fields):  buf[(flavor * Vs/2 + j) * 12 + (spin*3 + color)*2 + reim].
#include "tm_dslash.cuh"

namespace {

struct HaloGeom {
    int Vh;      // sites of one parity in the slab
    int Vs2;     // sites of one parity in a time slice
    int T;
};

template <int PREC> struct FaceReal { typedef float type; };
template <> struct FaceReal<8> { typedef double type; };

template <int PREC, int NF, int RECON>
__global__ void __launch_bounds__(128) halo_pack_kernel(typename FaceReal<PREC>::type *to_prev, typename FaceReal<PREC>::type *to_next,
                                                       const char *in, const char *gauge, HaloGeom g, int in_parity, int dagger)
{
    typedef typename PrecTraits<PREC>::real real;
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 2 * g.Vs2) return;
    const int which = tid / g.Vs2, j = tid - which * g.Vs2;          // 0: first slice -> previous slab, 1: last slice -> next slab
    const int site = which ? (g.T - 1) * g.Vs2 + j : j;
    const int lane = site & (TM_TILE - 1);
    // forward hop of the receiver (which = 0): projector sign +1 plain / -1 dagger; backward hop (which = 1): the opposite
    const bool lower = which == 0 ? !dagger : (dagger != 0);
    real u[18];
    if (which) {
        const size_t PB = (size_t)tm_tiles(g.Vh) * 4 * link_tile_bytes(PREC, RECON);
        load_link<PREC, RECON, false>(u, gauge + (size_t)in_parity * PB + link_site_off(PREC, RECON, site, 3), lane);
    }
#pragma unroll
    for (int f = 0; f < NF; f++) {
        real v[24], h[12];
        load_spinor<PREC, 0>(v, in + spinor_site_off(PREC, NF, site, f), lane);
#pragma unroll
        for (int i = 0; i < 12; i++) h[i] = lower ? v[12 + i] : v[i];
        typename FaceReal<PREC>::type *dst = (which ? to_next : to_prev) + ((size_t)f * g.Vs2 + j) * 12;
        if (which) {
            real gq[12];
            su3_mul<true>(gq, u, h);                                  // U_4(y)^dag h: the link belongs to the sender
#pragma unroll
            for (int i = 0; i < 12; i++) dst[i] = gq[i];
        } else {
#pragma unroll
            for (int i = 0; i < 12; i++) dst[i] = h[i];
        }
    }
}

template <int PREC, int NF, int RECON>
__global__ void __launch_bounds__(128) halo_apply_kernel(char *out, const typename FaceReal<PREC>::type *from_prev,
                                                        const typename FaceReal<PREC>::type *from_next, const char *gauge, HaloGeom g,
                                                        int parity, int dagger, double w_prev, double w_next, double alpha, double beta,
                                                        double scale, double coef, int twist_on)
{
    typedef typename PrecTraits<PREC>::real real;
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 2 * g.Vs2) return;
    const int which = tid / g.Vs2, j = tid - which * g.Vs2;          // 0: first slice, backward hop; 1: last slice, forward hop
    const int site = which ? (g.T - 1) * g.Vs2 + j : j;
    const int lane = site & (TM_TILE - 1);
    const bool lower = which == 1 ? !dagger : (dagger != 0);          // the half of the spinor the time hop feeds (tm_dslash.cuh)
    const real w = (real)(which ? w_next : w_prev);
    real u[18];
    if (which) {
        const size_t PB = (size_t)tm_tiles(g.Vh) * 4 * link_tile_bytes(PREC, RECON);
        load_link<PREC, RECON, false>(u, gauge + (size_t)parity * PB + link_site_off(PREC, RECON, site, 3), lane);
    }
    real acc[NF * 24];
#pragma unroll
    for (int i = 0; i < NF * 24; i++) acc[i] = 0;
#pragma unroll
    for (int f = 0; f < NF; f++) {
        const typename FaceReal<PREC>::type *src = (which ? from_next : from_prev) + ((size_t)f * g.Vs2 + j) * 12;
        real h[12], gq[12];
#pragma unroll
        for (int i = 0; i < 12; i++) h[i] = (real)src[i];
        if (which) su3_mul<false>(gq, u, h);                          // U_4(x) psi(x + t): the link is the receiver's own
#pragma unroll
        for (int i = 0; i < 12; i++) acc[24 * f + (lower ? 12 : 0) + i] = w * (which ? gq[i] : h[i]);
    }
    real lin[NF * 24];
    if (twist_on) {
#pragma unroll
        for (int f = 0; f < NF; f++)
            twist<NF>(lin + 24 * f, acc + 24 * f, acc + 24 * (NF - 1 - f), (real)(f == 0 ? alpha : -alpha), (real)beta, (real)scale);
    } else {
#pragma unroll
        for (int i = 0; i < NF * 24; i++) lin[i] = acc[i];
    }
#pragma unroll
    for (int f = 0; f < NF; f++) {
        char *os = out + spinor_site_off(PREC, NF, site, f);
        real v[24];
        load_spinor<PREC, 0>(v, os, lane);
#pragma unroll
        for (int i = 0; i < 24; i++) v[i] += (real)coef * lin[24 * f + i];
        store_spinor<PREC>(v, os, lane);
    }
}

HaloGeom geom_of(const tm_ctx *c)
{
    HaloGeom g;
    g.Vh = c->g.Vh;
    g.T = c->g.X[3];
    g.Vs2 = c->g.Vh / c->g.X[3];
    return g;
}

}  // namespace

#define TM_HALO_DISPATCH(CALL)                                                                          \
    do {                                                                                                \
        if (prec == 8) { if (nf == 1) { if (recon == 18) CALL(8, 1, 18); else if (recon == 12) CALL(8, 1, 12); else CALL(8, 1, 8); }   \
                         else { if (recon == 18) CALL(8, 2, 18); else if (recon == 12) CALL(8, 2, 12); else CALL(8, 2, 8); } }          \
        else if (prec == 4) { if (nf == 1) { if (recon == 18) CALL(4, 1, 18); else if (recon == 12) CALL(4, 1, 12); else CALL(4, 1, 8); } \
                         else { if (recon == 18) CALL(4, 2, 18); else if (recon == 12) CALL(4, 2, 12); else CALL(4, 2, 8); } }          \
        else { if (nf == 1) { if (recon == 18) CALL(2, 1, 18); else if (recon == 12) CALL(2, 1, 12); else CALL(2, 1, 8); }               \
               else { if (recon == 18) CALL(2, 2, 18); else if (recon == 12) CALL(2, 2, 12); else CALL(2, 2, 8); } }                    \
    } while (0)

cudaError_t tm_launch_halo_pack(const tm_field *in, const tm_gauge *gg, int out_parity, int dagger, void *to_prev, void *to_next, cudaStream_t s)
{
    const HaloGeom g = geom_of(in->ctx);
    const int prec = in->prec, nf = in->nf, recon = gg->recon;
    const int threads = 128, blocks = (2 * g.Vs2 + threads - 1) / threads;
    const char *ip = static_cast<const char *>(in->ptr), *gp = static_cast<const char *>(gg->ptr);
#define TM_HP(P, N, R)                                                                                                     \
    halo_pack_kernel<P, N, R><<<blocks, threads, 0, s>>>(static_cast<FaceReal<P>::type *>(to_prev), static_cast<FaceReal<P>::type *>(to_next), \
                                                         ip, gp, g, 1 - out_parity, dagger)
    TM_HALO_DISPATCH(TM_HP);
#undef TM_HP
    return cudaGetLastError();
}

cudaError_t tm_launch_halo_apply(tm_field *out, const void *from_prev, const void *from_next, const tm_gauge *gg, int parity, int dagger,
                                 double w_prev, double w_next, double alpha, double beta, double scale, double coef, int twist_on, cudaStream_t s)
{
    const HaloGeom g = geom_of(out->ctx);
    const int prec = out->prec, nf = out->nf, recon = gg->recon;
    const int threads = 128, blocks = (2 * g.Vs2 + threads - 1) / threads;
    char *op = static_cast<char *>(out->ptr);
    const char *gp = static_cast<const char *>(gg->ptr);
#define TM_HA(P, N, R)                                                                                                               \
    halo_apply_kernel<P, N, R><<<blocks, threads, 0, s>>>(op, static_cast<const FaceReal<P>::type *>(from_prev),                     \
                                                          static_cast<const FaceReal<P>::type *>(from_next), gp, g, parity, dagger,   \
                                                          w_prev, w_next, alpha, beta, scale, coef, twist_on)
    TM_HALO_DISPATCH(TM_HA);
#undef TM_HA
    return cudaGetLastError();
}

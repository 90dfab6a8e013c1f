// tm_twist.cu -- the local twist alone:  out = R in,  R^-1 in,  R^dag in  or  R^dag^-1 in  on one parity field
// (R = 1 + i a gamma5 tau3 + b tau1, C2).  The dslash kernels apply R or R^-1 in their epilogue; this
// kernel covers the places where the twist stands in front of a hopping term: the adjoint of the symmetric
// operator (M^_sym^dag = 1 - kappa^2 D^dag R^dag^-1 D^dag R^dag^-1) and the right-hand sides of Eq. 2.2 / 2.3
// (b_e + kappa D_eo R_oo^-1 b_o).  One thread per site, every flavor of the site; pure streaming.
#include "tm_dslash.cuh"

template <int PREC, int NF>
__global__ void __launch_bounds__(128) tm_twist_kernel(char *out, const char *in, int Vh, double alpha, double beta, double scale)
{
    typedef typename PrecTraits<PREC>::real real;
    const int site = blockIdx.x * blockDim.x + threadIdx.x;
    if (site >= Vh) return;
    const int lane = site & (TM_TILE - 1);
    const size_t off = spinor_site_off(PREC, NF, site, 0);
    real v[NF * 24], w[NF * 24];
#pragma unroll
    for (int f = 0; f < NF; f++) load_spinor<PREC, 0>(v + 24 * f, in + off + f * spinor_tile_bytes(PREC), lane);
#pragma unroll
    for (int f = 0; f < NF; f++)
        twist<NF>(w + 24 * f, v + 24 * f, v + 24 * (NF - 1 - f), f == 0 ? (real)alpha : (real)-alpha, (real)beta, (real)scale);
#pragma unroll
    for (int f = 0; f < NF; f++) store_spinor<PREC>(w + 24 * f, out + off + f * spinor_tile_bytes(PREC), lane);
}

cudaError_t tm_launch_twist(const tm_field *out, const tm_field *in, double alpha, double beta, double scale, cudaStream_t s)
{
    const int Vh = out->ctx->g.Vh, threads = 128, blocks = (Vh + threads - 1) / threads;
    char *o = static_cast<char *>(out->ptr);
    const char *i = static_cast<const char *>(in->ptr);
#define TM_TW(P, N) tm_twist_kernel<P, N><<<blocks, threads, 0, s>>>(o, i, Vh, alpha, beta, scale)
    if (out->prec == 8) { if (out->nf == 1) TM_TW(8, 1); else TM_TW(8, 2); }
    else if (out->prec == 4) { if (out->nf == 1) TM_TW(4, 1); else TM_TW(4, 2); }
    else { if (out->nf == 1) TM_TW(2, 1); else TM_TW(2, 2); }
#undef TM_TW
    return cudaGetLastError();
}

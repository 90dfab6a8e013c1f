// tm_noalloc.cu -- Re <x, y> (the reduction of the mixed-precision CG) for callers that may not allocate:
// code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  tm_blas.cu keeps the per-block partial
// sums of its reductions in a cudaMalloc'ed buffer on the context, grown on demand; this variant keeps them in a file-scope
// __device__ array of fixed size instead, so the entry point (tm_field_redot_noalloc, include/tm.h) calls no cudaMalloc, no
// cudaFree and no allocating library routine -- and accepts at most TM_NOALLOC_MAX_SITES sites per parity.
//
// The array costs TM_NOALLOC_MAX_BLOCKS x 8 bytes = 512 KiB of device memory on EVERY GPU that loads the library, until the
// process exits.  Every call on a device shares it and it keeps the last call's contents: a call overwrites partial[0 .. blocks)
// before it reads them and reads nothing beyond, so nothing has to start at zero -- but two calls that overlap on the GPU
// (different contexts / streams of one device, or two host threads) race on it.  Calls on one context stream are ordered.
//
// Same arithmetic and the same summation order as redot_kernel / final_sum_kernel of tm_blas.cu (one thread per site in
// double, warp shuffle tree, warps of a block in order, then 256 strided slices and a fixed tree): the two paths agree bit for bit.
#include <mutex>

#include "tm_internal.h"
#include "tm_layout.cuh"

// In host code this name is a host-side stand-in, NOT a device address: only cudaGetSymbolAddress (scratch_of below) turns it
// into a pointer a kernel may use.
static __device__ __align__(256) double tm_noalloc_scratch[TM_NOALLOC_MAX_BLOCKS];

namespace {

constexpr int BT = TM_NOALLOC_BLOCK;          // threads (= sites) per block
constexpr int MAX_DEVICES = 64;

template <int P, int NF>
__global__ void __launch_bounds__(BT) redot_noalloc_kernel(const char *x, const char *y, int Vh, double *partial)
{
    __shared__ double sh[BT / 32];
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
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0;
#pragma unroll
        for (int w = 0; w < BT / 32; w++) t += sh[w];
        partial[blockIdx.x] = t;
    }
}

// out[0] = partial[0] + ... + partial[n - 1] in a fixed order (one block)
__global__ void __launch_bounds__(256) sum_noalloc_kernel(const double *partial, int n, double *out)
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

// Set-up, once per device and with that device current: the device address of the array on THAT device (every device
// that loads the module has its own copy at its own address).
std::mutex g_mu;
double *g_scratch[MAX_DEVICES] = {};

cudaError_t scratch_of(int device, double **out)
{
    if (device < 0 || device >= MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch[device]) {
        int cur = -1;
        cudaError_t e = cudaGetDevice(&cur);
        if (e != cudaSuccess) return e;
        if (cur != device && (e = cudaSetDevice(device)) != cudaSuccess) return e;
        double *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, tm_noalloc_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_scratch[device] = p;
    }
    *out = g_scratch[device];
    return cudaSuccess;
}

}  // namespace

// *dev_out (DEVICE) = Re <x, y>; x, y checked by the caller (tm_api.cu: same context, precision, flavors, Vh within the
// maximum).  Two launches on the context stream, nothing allocated, nothing synchronised.
cudaError_t tm_noalloc_redot(const tm_field *x, const tm_field *y, double *dev_out)
{
    tm_ctx *c = x->ctx;
    const int Vh = c->g.Vh;
    if (Vh <= 0 || (long)Vh > (long)TM_NOALLOC_MAX_SITES) return cudaErrorInvalidValue;
    const int blocks = (Vh + BT - 1) / BT;
    double *scratch = nullptr;
    cudaError_t e = scratch_of(c->device, &scratch);
    if (e != cudaSuccess) return e;
    int cur = -1;
    if ((e = cudaGetDevice(&cur)) != cudaSuccess) return e;
    if (cur != c->device && (e = cudaSetDevice(c->device)) != cudaSuccess) return e;
    const char *xp = static_cast<const char *>(x->ptr), *yp = static_cast<const char *>(y->ptr);
#define TM_DOT(P, N) redot_noalloc_kernel<P, N><<<blocks, BT, 0, c->stream>>>(xp, yp, Vh, scratch)
    if (x->prec == 8) { if (x->nf == 1) TM_DOT(8, 1); else TM_DOT(8, 2); }
    else if (x->prec == 4) { if (x->nf == 1) TM_DOT(4, 1); else TM_DOT(4, 2); }
    else { if (x->nf == 1) TM_DOT(2, 1); else TM_DOT(2, 2); }
#undef TM_DOT
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    sum_noalloc_kernel<<<1, 256, 0, c->stream>>>(scratch, blocks, dev_out);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    c->launches++;
    c->last_kernel = "redot_noalloc";
    // multi-GPU: the caller's all-reduce hook (tm_set_allreduce) sums the device word over the ranks, in stream order
    if (c->allreduce && c->allreduce(dev_out, 1, static_cast<void *>(c->stream), c->allreduce_user) != 0) return cudaErrorUnknown;
    return cudaSuccess;
}

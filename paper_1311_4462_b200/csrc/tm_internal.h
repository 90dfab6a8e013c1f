// tm_internal.h -- private structures shared by the C-ABI layer (tm_api.cu) and the kernel launchers.
// Device layout (row a1; addressing helpers in tm_layout.cuh): tiles of 32 consecutive
// checkerboard sites, inside a tile one 512-byte plane per 128-bit chunk
//   spinor, one parity : [tile][flavor][plane][32]
//        fp64: 12 planes of double2 (one complex each, index spin*3+color)
//        fp32:  6 planes of float4  (two complex each)
//        half:  3 planes of 8 x int16 + one 128-byte plane of float norms
//   gauge : [parity][tile][mu][plane][32]; a link's reals r = (row*3+col)*2+reim are cut into planes
//        fp64: recon/2 planes of double2
//        fp32: 18 -> 4 x float4 + 1 x float2 ; 12 -> 3 x float4
//        half: 18 -> 2 x int4(8 x int16) + 1 x int(2 x int16) ; 12 -> 1 x int4 + 1 x int2
//        8-real (tm_layout.cuh: rebuild_from8): 4 x double2 / 2 x float4 / 1 x int4
//   the [parity] block holds U_mu(x) for the sites x of that parity.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

#include <atomic>
#include <vector>

#include "../../include/tm.h"

struct TmGeom {
    int X[4];
    int Xh;      // X/2
    int Vh;      // V/2
    long V;
};

struct tm_ctx {
    TmGeom g;
    int device;
    cudaStream_t stream;
    long launches;
    const char *last_kernel;
    int path;    // 0 auto, 1 generic only
    int pf_dist; // tm_set_tuning("prefetch_blocks")
    int stage;   // tm_set_tuning("stage_links"): -1 library default, 0 direct loads, 1 links staged through shared memory
    int block_threads;   // tm_set_tuning("block_threads"): 0 library default, else 32 / 64 / 128
    int pdl;             // tm_set_tuning("pdl"): 1 (default) = fused kernels are launched with programmatic stream serialization, 0 = plain launches
    int tile_kernel;     // tm_set_tuning("tile_kernel"): -1 library default (on where the geometry allows), 0 off, 1 on
    int z_chunks;        // tm_set_tuning("z_chunks"): -1 library default (from the L2 working set), else the number of z-chunks
    int sm_count;
    int basis_on;         // tm_set_host_basis: host spinors are in another spin basis, psi_device = S psi_host
    double basis[32];     // S, row-major [4][4][re, im]
    void *staging;        // device staging for upload / download
    // asynchronous upload / download (tm_field_upload_cb_async / tm_field_download_cb_async): one copy stream per direction with
    // its own staging, ordered against the compute stream by events
    cudaStream_t up_stream, down_stream;
    cudaEvent_t ev_compute, ev_up, ev_down;
    void *up_staging, *down_staging;
    size_t up_bytes, down_bytes;
    bool async_ready;
    int open_mask;        // tm_set_open_dirs: bit mu set = the fused kernels drop the mu hops that leave the sub-lattice (tm_halo.cu adds them)
    unsigned *halo_counter;   // device word: blocks of the running halo_pack kernel that have finished (flag signalling)
    tm_allreduce_fn allreduce;   // tm_set_allreduce: sums a device word over the ranks (NULL: one GPU)
    void *allreduce_user;
    std::vector<tm_field *> cg_ws;   // work fields of tm_invert_cg, kept between solves (freed by tm_cg_release / tm_finalize)
    double *cgs;          // inner CG scalars on the device: [0], [1] |r|^2 (ping-pong), [2] <p, A p>
    double *cgs_host;     // pinned host ring the scalars are copied to: 2 x 3 doubles
    cudaEvent_t cg_ev[2]; // one event per ring slot
    double *red;          // reduction scratch of tm_blas.cu: [0] result, [1..] per-block partial sums
    size_t red_n;
    size_t staging_bytes;
    bool timing;          // tm_timing_enable
    bool timing_chain;    // tm_timing_enable(ctx, 2): one event BETWEEN consecutive launches (a launch's start is its predecessor's stop)
    struct TimedLaunch { cudaEvent_t start, stop; const char *name; bool own_start; };
    std::vector<TimedLaunch> timed;
};

struct tm_field {
    tm_ctx *ctx;
    int prec;    // 8 / 4 / 2
    int nf;      // 1 / 2
    void *ptr;
    size_t bytes;
    bool owns;
};

struct tm_gauge {
    tm_ctx *ctx;
    int prec;
    int recon;
    void *ptr;
    size_t bytes;
};


// Division of a site index (< 2^31) by a lattice extent d >= 2 without the integer-division sequence:
// q = umulhi(n, m) >> sh with m = floor(2^(31+l) / d) + 1, l = ceil(log2 d), sh = l - 1 (exact for every n < 2^31).
struct TmFastDiv {
    unsigned m;
    int sh;
    int d;
};
static inline TmFastDiv tm_fastdiv(int d)
{
    TmFastDiv f;
    int l = 0;
    while ((1LL << l) < d) l++;
    f.m = (unsigned)(((1ULL << (31 + l)) / (unsigned long long)d) + 1ULL);
    f.sh = l - 1;
    f.d = d;
    return f;
}
#ifdef __CUDACC__
__device__ __forceinline__ int tm_div(int n, const TmFastDiv &f) { return (int)(__umulhi((unsigned)n, f.m) >> f.sh); }
#endif

// Arguments of one fused dslash launch.  Coefficients are formed in double on the host (reading C10-ii)
// and cast to the kernel's arithmetic type on the device.
struct DslashArgs {
    void *out;
    const void *in;
    const void *x;
    const void *gauge;
    int X, Y, Z, T, Xh, Vh;
    TmFastDiv dXh, dY, dZ;   // site decode
    int parity;          // parity of the output sites
    double alpha;        // local twist, flavor 0:  w = scale * (v + i alpha gamma5 v + beta v_otherflavor)
    double beta;
    double scale;
    int pdl;             // launch with programmatic stream serialization (the kernels call griddepcontrol themselves)
    double alpha_in, beta_in, scale_in;   // TWIN kernels: the twist applied to the input sites (same form as alpha / beta / scale)
    double kappa;        // REC
    double kappa2;       // A-xpay, B
    double tbound;       // +-1 (0 when the time direction is decomposed), multiplies the time hop that wraps
    float wrap_y, wrap_z;   // weight of the y / z hop that wraps: 1, or 0 when that direction is decomposed (tm_set_open_dirs)
    int block_threads;   // threads per block (= sites per block)
    int pf_dist;         // L2 prefetch distance in thread blocks (0 = off): block b prefetches the tile of block b + pf_dist
    // z-chunked traversal (tm_virtual_block): thread blocks walk the lattice chunk by chunk of Z / nzc z-planes, all time slices
    // of a chunk before the next chunk, so that the three time slices of input spinor a block range re-reads fit the L2
    int nzc;             // number of z-chunks (1 = plain index order)
    int bpz;             // thread blocks per (time slice, chunk)
    TmFastDiv dbpc, dbpz;   // division by bpz * T and by bpz
};
#ifdef __CUDACC__
// The block of sites that thread block b works on.  nzc == 1: b itself.  Otherwise b counts (chunk, t, block within the chunk's
// part of slice t), while site order is (t, z, y, x): the virtual block is (t * nzc + chunk) * bpz + w.
__device__ __forceinline__ int tm_virtual_block(const DslashArgs &a, int b)
{
    if (a.nzc <= 1) return b;
    const int c = tm_div(b, a.dbpc);
    const int r = b - c * a.dbpc.d;
    const int t = tm_div(r, a.dbpz);
    const int w = r - t * a.bpz;
    return (t * a.nzc + c) * a.bpz + w;
}
#endif

// Kernels that stage more than 48 KB of shared memory need cudaFuncAttributeMaxDynamicSharedMemorySize raised; the
// attribute is per DEVICE, so it is remembered per (instantiation, device id) in a bit mask, not per process.
template <class K>
inline cudaError_t tm_raise_smem(K kernel, std::atomic<unsigned long long> &done)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const unsigned long long bit = 1ULL << (dev & 63);
    if (dev < 64 && (done.load(std::memory_order_relaxed) & bit)) return cudaSuccess;
    e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    if (e == cudaSuccess && dev < 64) done.fetch_or(bit, std::memory_order_relaxed);
    return e;
}

// Launch of a fused dslash kernel.  pdl != 0: with the programmatic-stream-serialization attribute, so that the launch is set up on the
// GPU while the previous kernel of the stream still runs (every fused kernel executes griddepcontrol.wait before its first access to a
// field and none triggers its dependents early: execution order = that of plain launches, tm_stream.cuh).
template <class... KArgs, class... Args>
inline cudaError_t tm_launch_kernel(void (*kernel)(KArgs...), int pdl, unsigned grid, unsigned block, size_t smem, cudaStream_t s, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid, 1, 1);
    cfg.blockDim = dim3(block, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// kernel launchers (one translation unit per precision x flavor count)
typedef cudaError_t (*tm_launch_fn)(const DslashArgs &, cudaStream_t);
struct TmKernelEntry {
    tm_launch_fn fn;
    const char *name;
};
// index: [recon 18 / 12 / 8 -> 0 / 1 / 2][kt 0..3][dagger 0..1][staged 0..1]  (8-real: scalar kernels only)
const TmKernelEntry *tm_generic_table(int prec, int nf);

// out = scale (1 + i alpha gamma5 tau3 + beta tau1) in, site by site (tm_twist.cu)
cudaError_t tm_launch_twist(const tm_field *out, const tm_field *in, double alpha, double beta, double scale, cudaStream_t s);

// vector operations of the CG (tm_blas.cu); the ones that return a sum synchronise the stream
cudaError_t tm_blas_axpbyz(tm_field *z, double a, const tm_field *x, double b, const tm_field *y, double *norm2);
cudaError_t tm_blas_redot(const tm_field *x, const tm_field *y, double *out);
cudaError_t tm_blas_cg_update(tm_field *x, tm_field *r, const tm_field *p, const tm_field *Ap, double a, double *rr);
// the same with the scalars read from / left in DEVICE memory (no stream synchronisation): the inner CG loop
cudaError_t tm_blas_axpbyz_dev(tm_field *z, double a, const tm_field *x, double b, const tm_field *y, double *norm2,
                               const double *bnum, const double *bden);
cudaError_t tm_blas_redot_dev(const tm_field *x, const tm_field *y, double *out, double *dev_out);
cudaError_t tm_blas_cg_update_dev(tm_field *x, tm_field *r, const tm_field *p, const tm_field *Ap, double a, double *rr,
                                  const double *anum, const double *aden, double *dev_rr);

// Re <x, y> with its scratch in a fixed __device__ array (tm_noalloc.cu): no allocation, result left in DEVICE memory
#define TM_NOALLOC_BLOCK 128
#define TM_NOALLOC_MAX_BLOCKS ((int)(TM_NOALLOC_MAX_SITES / TM_NOALLOC_BLOCK))
cudaError_t tm_noalloc_redot(const tm_field *x, const tm_field *y, double *dev_out);

// surface kernels of the domain decomposition (tm_halo.cu); dir = 1 (y), 2 (z), 3 (t)
cudaError_t tm_launch_halo_pack(const tm_field *in, const tm_gauge *g, int out_parity, int dagger, int dir, void *to_prev, void *to_next,
                                unsigned *flag_prev, unsigned *flag_next, unsigned epoch, unsigned *counter, cudaStream_t s);
cudaError_t tm_launch_halo_apply(tm_field *out, const void *from_prev, const void *from_next, const tm_gauge *g, int parity, int dagger, int dir,
                                 double w_prev, double w_next, double alpha, double beta, double scale, double coef, int twist_on,
                                 const unsigned *wait_prev, const unsigned *wait_next, unsigned epoch, cudaStream_t s);

// pack / unpack (tm_pack.cu)
// (both apply the context's host spin basis: S on the way in, S^dag on the way out)
// host_prec: 8 = double arrays (the canonical form), 4 = float arrays
cudaError_t tm_pack_spinor(const tm_field *f, int parity, const void *dev_src, int host_prec, bool src_is_cb, cudaStream_t s);
cudaError_t tm_unpack_spinor(const tm_field *f, int parity, void *dev_dst, int host_prec, bool dst_is_cb, cudaStream_t s);
cudaError_t tm_pack_gauge(const tm_gauge *g, const double *dev_src, cudaStream_t s);

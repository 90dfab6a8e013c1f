// tm_halo.cu -- domain decomposition in y, z and t ("redesign QUDA packing routines
// to properly take into account the fifth flavor dimension when gathering boundary-spinor sites in non-temporal lattice
// directions", :134 multi-GPU runs).  The lattice is cut into sub-lattices, one per GPU; the fused dslash kernels run on the
// sub-lattice with the hops that leave it in a cut direction switched off (tm_set_open_dirs); this file supplies the two
// surface kernels around the exchange, for one cut direction DIR = 1 (y), 2 (z), 3 (t) per launch:
//   halo_pack  : spin-projected half-spinors (12 reals per site AND FLAVOR: the doublet's face carries the flavor index) of the
//                first slice x_DIR = 0 (for the previous sub-lattice's forward hops) and U_DIR^dag times the projected
//                half-spinors of the last slice (for the next one's backward hops: the link lives with the sender).
//                A face of a non-temporal direction is a strided set of sites of the tiled layout (face_site below).
//   halo_apply : adds the missing hops to the boundary sites of the kernel's output.  Every fused epilogue is affine in the
//                hopping sum, so out += coef * [twist](acc_surface) completes A, A-xpay, B, REC and the twist-free forms, and
//                the completions of different directions commute.
// Face site j = checkerboard order of the face's sites (x fastest, then the uncut coordinates): the boundary site and its
// neighbour across the cut have the same j (they differ in x_DIR only; the x-offset of the checkerboard flips twice).
// Buffers hold double (fp64 fields) or float (fp32 and half fields):  buf[(flavor * Vf + j) * 12 + (spin*3 + color)*2 + reim].
// Signalling (optional): with peer-mapped receive buffers the pack kernel's stores ARE the transfer; its last block then stores
// the epoch to the neighbours' flag words (release, system scope) and halo_apply spins on its own flag words (acquire).
#include "tm_dslash.cuh"

namespace {

struct HaloGeom {
    int Vh;      // sites of one parity in the sub-lattice
    int Vf;      // sites of one parity in a face of this direction
    int L;       // local extent in the cut direction
    int A;       // sites of one parity per unit step of the cut coordinate (Xh for y, Xh Y for z, Xh Y Z for t)
    TmFastDiv dA;
};

// checkerboard index of face site j in slice s (0 or L - 1) of the cut direction
TM_DEV int face_site(const HaloGeom &g, int j, int s)
{
    const int jh = tm_div(j, g.dA), jl = j - jh * g.A;
    return jl + g.A * (s + g.L * jh);
}

template <int PREC> struct FaceReal { typedef float type; };
template <> struct FaceReal<8> { typedef double type; };

TM_DEV void flag_release(unsigned *p, unsigned v) { asm volatile("st.release.sys.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory"); }
TM_DEV unsigned flag_acquire(const unsigned *p)
{
    unsigned v;
    asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// the half-spinor a hop of direction DIR with projector sign SGN carries
template <int DIR, typename real>
TM_DEV void project_dir(real *h, const real *v, int sgn)
{
    if constexpr (DIR == 3) {
#pragma unroll
        for (int i = 0; i < 12; i++) h[i] = sgn > 0 ? v[12 + i] : v[i];
    } else {
        if (sgn > 0) project<DIR, +1>(h, v);
        else project<DIR, -1>(h, v);
    }
}

template <int PREC, int NF, int RECON, int DIR>
__global__ void __launch_bounds__(128) halo_pack_kernel(typename FaceReal<PREC>::type *to_prev, typename FaceReal<PREC>::type *to_next,
                                                       const char *in, const char *gauge, HaloGeom g, int in_parity, int dagger,
                                                       unsigned *flag_prev, unsigned *flag_next, unsigned epoch, unsigned *counter)
{
    typedef typename PrecTraits<PREC>::real real;
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid < 2 * g.Vf) {
        const int which = tid / g.Vf, j = tid - which * g.Vf;       // 0: first slice -> previous, 1: last slice -> next
        const int site = face_site(g, j, which ? g.L - 1 : 0);
        const int lane = site & (TM_TILE - 1);
        // forward hop of the receiver (which = 0): projector sign +1 plain / -1 dagger; backward hop (which = 1): the opposite
        const int sgn = (which == 0) == (dagger == 0) ? +1 : -1;
        real u[18];
        if (which) {
            const size_t PB = (size_t)tm_tiles(g.Vh) * 4 * link_tile_bytes(PREC, RECON);
            load_link<PREC, RECON, false>(u, gauge + (size_t)in_parity * PB + link_site_off(PREC, RECON, site, DIR), lane);
        }
#pragma unroll
        for (int f = 0; f < NF; f++) {
            real v[24], h[12];
            load_spinor<PREC, 0>(v, in + spinor_site_off(PREC, NF, site, f), lane);
            project_dir<DIR>(h, v, sgn);
            typename FaceReal<PREC>::type *dst = (which ? to_next : to_prev) + ((size_t)f * g.Vf + j) * 12;
            if (which) {
                real gq[12];
                su3_mul<true>(gq, u, h);                              // U_DIR(y)^dag h: the link belongs to the sender
#pragma unroll
                for (int i = 0; i < 12; i++) dst[i] = gq[i];
            } else {
#pragma unroll
                for (int i = 0; i < 12; i++) dst[i] = h[i];
            }
        }
    }
    if (flag_prev || flag_next) {          // the last block to finish publishes the epoch (all blocks' stores are visible first)
        __threadfence_system();
        __syncthreads();
        if (threadIdx.x == 0) {
            const unsigned done = atomicAdd(counter, 1u);
            if (done == gridDim.x - 1) {
                *counter = 0;
                __threadfence_system();
                if (flag_prev) flag_release(flag_prev, epoch);
                if (flag_next) flag_release(flag_next, epoch);
            }
        }
    }
}

template <int PREC, int NF, int RECON, int DIR>
__global__ void __launch_bounds__(128) halo_apply_kernel(char *out, const typename FaceReal<PREC>::type *from_prev,
                                                        const typename FaceReal<PREC>::type *from_next, const char *gauge, HaloGeom g,
                                                        int parity, int dagger, double w_prev, double w_next, double alpha, double beta,
                                                        double scale, double coef, int twist_on, const unsigned *wait_prev,
                                                        const unsigned *wait_next, unsigned epoch)
{
    typedef typename PrecTraits<PREC>::real real;
    if (wait_prev || wait_next) {          // the faces are written by the neighbours' pack kernels: wait for this epoch's signal
        if (threadIdx.x == 0) {
            if (wait_prev) while ((int)(flag_acquire(wait_prev) - epoch) < 0) { }
            if (wait_next) while ((int)(flag_acquire(wait_next) - epoch) < 0) { }
        }
        __syncthreads();
    }
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 2 * g.Vf) return;
    const int which = tid / g.Vf, j = tid - which * g.Vf;            // 0: first slice, backward hop; 1: last slice, forward hop
    const int site = face_site(g, j, which ? g.L - 1 : 0);
    const int lane = site & (TM_TILE - 1);
    const int sgn = (which == 1) == (dagger == 0) ? +1 : -1;          // projector sign of the hop being added (tm_dslash.cuh: hop)
    const real w = (real)(which ? w_next : w_prev);
    real u[18];
    if (which) {
        const size_t PB = (size_t)tm_tiles(g.Vh) * 4 * link_tile_bytes(PREC, RECON);
        load_link<PREC, RECON, false>(u, gauge + (size_t)parity * PB + link_site_off(PREC, RECON, site, DIR), lane);
    }
    real acc[NF * 24];
#pragma unroll
    for (int i = 0; i < NF * 24; i++) acc[i] = 0;
#pragma unroll
    for (int f = 0; f < NF; f++) {
        const typename FaceReal<PREC>::type *src = (which ? from_next : from_prev) + ((size_t)f * g.Vf + j) * 12;
        real h[12], gq[12];
#pragma unroll
        for (int i = 0; i < 12; i++) h[i] = (real)__ldcg(src + i);    // L2: the writer may be another GPU
        if (which) su3_mul<false>(gq, u, h);                          // U_DIR(x) psi(x + dir): the link is the receiver's own
        else {
#pragma unroll
            for (int i = 0; i < 12; i++) gq[i] = h[i];
        }
        if (sgn > 0) reconstruct_acc<DIR, +1>(acc + 24 * f, gq, w);
        else reconstruct_acc<DIR, -1>(acc + 24 * f, gq, w);
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

HaloGeom geom_of(const tm_ctx *c, int dir)
{
    HaloGeom g;
    g.Vh = c->g.Vh;
    g.L = c->g.X[dir];
    g.Vf = c->g.Vh / g.L;
    g.A = c->g.Xh;
    for (int d = 1; d < dir; d++) g.A *= c->g.X[d];
    g.dA = tm_fastdiv(g.A);
    return g;
}

}  // namespace

#define TM_HALO_RECON(CALL, P, N, D)                                                                     \
    do { if (recon == 18) CALL(P, N, 18, D); else if (recon == 12) CALL(P, N, 12, D); else CALL(P, N, 8, D); } while (0)
#define TM_HALO_NF(CALL, P, D) do { if (nf == 1) TM_HALO_RECON(CALL, P, 1, D); else TM_HALO_RECON(CALL, P, 2, D); } while (0)
#define TM_HALO_PREC(CALL, D)                                                                            \
    do { if (prec == 8) TM_HALO_NF(CALL, 8, D); else if (prec == 4) TM_HALO_NF(CALL, 4, D); else TM_HALO_NF(CALL, 2, D); } while (0)
#define TM_HALO_DISPATCH(CALL)                                                                           \
    do { if (dir == 1) TM_HALO_PREC(CALL, 1); else if (dir == 2) TM_HALO_PREC(CALL, 2); else TM_HALO_PREC(CALL, 3); } while (0)

cudaError_t tm_launch_halo_pack(const tm_field *in, const tm_gauge *gg, int out_parity, int dagger, int dir, void *to_prev, void *to_next,
                                unsigned *flag_prev, unsigned *flag_next, unsigned epoch, unsigned *counter, cudaStream_t s)
{
    const HaloGeom g = geom_of(in->ctx, dir);
    const int prec = in->prec, nf = in->nf, recon = gg->recon;
    const int threads = 128, blocks = (2 * g.Vf + threads - 1) / threads;
    const char *ip = static_cast<const char *>(in->ptr), *gp = static_cast<const char *>(gg->ptr);
#define TM_HP(P, N, R, D)                                                                                                       \
    halo_pack_kernel<P, N, R, D><<<blocks, threads, 0, s>>>(static_cast<FaceReal<P>::type *>(to_prev), static_cast<FaceReal<P>::type *>(to_next), \
                                                            ip, gp, g, 1 - out_parity, dagger, flag_prev, flag_next, epoch, counter)
    TM_HALO_DISPATCH(TM_HP);
#undef TM_HP
    return cudaGetLastError();
}

cudaError_t tm_launch_halo_apply(tm_field *out, const void *from_prev, const void *from_next, const tm_gauge *gg, int parity, int dagger, int dir,
                                 double w_prev, double w_next, double alpha, double beta, double scale, double coef, int twist_on,
                                 const unsigned *wait_prev, const unsigned *wait_next, unsigned epoch, cudaStream_t s)
{
    const HaloGeom g = geom_of(out->ctx, dir);
    const int prec = out->prec, nf = out->nf, recon = gg->recon;
    const int threads = 128, blocks = (2 * g.Vf + threads - 1) / threads;
    char *op = static_cast<char *>(out->ptr);
    const char *gp = static_cast<const char *>(gg->ptr);
#define TM_HA(P, N, R, D)                                                                                                            \
    halo_apply_kernel<P, N, R, D><<<blocks, threads, 0, s>>>(op, static_cast<const FaceReal<P>::type *>(from_prev),                  \
                                                             static_cast<const FaceReal<P>::type *>(from_next), gp, g, parity, dagger, \
                                                             w_prev, w_next, alpha, beta, scale, coef, twist_on, wait_prev, wait_next, epoch)
    TM_HALO_DISPATCH(TM_HA);
#undef TM_HA
    return cudaGetLastError();
}

// tm_dslash.cuh -- the generic fused twisted-mass dslash kernel (rows a2-a9 of DESIGN.md).
// One thread per output site (both flavors of a doublet); direct 128-bit read-only loads, neighbour reuse through L1/L2.
// Works for every even lattice with extents >= 4.  The production path for fp64; fp32 and half run the packed
// kernels of tm_dslash_f2.cuh and fall back to this one only for combinations those do not cover.
//
// gamma basis (C5):  gamma_k = [[0, i s_k], [-i s_k, 0]],  gamma_4 = diag(1,1,-1,-1),  gamma_5 swaps
// the upper and lower two spin components.  With sgn = +1 for (1 - gamma_mu), -1 for (1 + gamma_mu):
//   spatial:  h = psi_u - sgn * i s_k psi_l ;  (1 -+ gamma_k) psi = [h ; sgn * i s_k h]
//   time   :  (1 - gamma_4) psi = [0 ; 2 psi_l],  (1 + gamma_4) psi = [2 psi_u ; 0]   -> only half the spinor is read
#pragma once
#include "tm_internal.h"
#include "tm_layout.cuh"
#include "tm_stream.cuh"

// ---- spin projection (a3): 24 -> 12 reals -----------------------------------------------------------
template <int MU, int SGN, typename real>
TM_DEV void project(real *h, const real *v)
{
    const real *u = v, *l = v + 12;     // [spin 0..1][color][reim]
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int a = 2 * c, b = 6 + 2 * c;     // spin 0 / spin 1 of the half
        if constexpr (MU == 0) {                // i s_1 v = (i v_1, i v_0)
            h[a] = u[a] + SGN * l[b + 1];
            h[a + 1] = u[a + 1] - SGN * l[b];
            h[b] = u[b] + SGN * l[a + 1];
            h[b + 1] = u[b + 1] - SGN * l[a];
        } else if constexpr (MU == 1) {         // i s_2 v = (v_1, -v_0)
            h[a] = u[a] - SGN * l[b];
            h[a + 1] = u[a + 1] - SGN * l[b + 1];
            h[b] = u[b] + SGN * l[a];
            h[b + 1] = u[b + 1] + SGN * l[a + 1];
        } else if constexpr (MU == 2) {         // i s_3 v = (i v_0, -i v_1)
            h[a] = u[a] + SGN * l[a + 1];
            h[a + 1] = u[a + 1] - SGN * l[a];
            h[b] = u[b] - SGN * l[b + 1];
            h[b + 1] = u[b + 1] + SGN * l[b];
        }
    }
}

// ---- color multiply (a5): g = U h (forward) or U^dag h (backward), two spin components -------------
template <bool ADJ, typename real>
TM_DEV void su3_mul(real *g, const real *u, const real *h)
{
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
        for (int c = 0; c < 3; c++) {
            real re, im;
#pragma unroll
            for (int d = 0; d < 3; d++) {
                const real hr = h[6 * s + 2 * d], hi = h[6 * s + 2 * d + 1];
                // explicit FMA chains (4 per complex multiply-add); ADJ: conj(U[d][c])
                const real ur = ADJ ? u[2 * (3 * d + c)] : u[2 * (3 * c + d)];
                const real ui = ADJ ? -u[2 * (3 * d + c) + 1] : u[2 * (3 * c + d) + 1];
                if (d == 0) {
                    re = ur * hr;
                    im = ur * hi;
                } else {
                    re = tm_fma(ur, hr, re);
                    im = tm_fma(ur, hi, im);
                }
                re = tm_fma(-ui, hi, re);
                im = tm_fma(ui, hr, im);
            }
            g[6 * s + 2 * c] = re;
            g[6 * s + 2 * c + 1] = im;
        }
}

// ---- spin reconstruction + accumulate (a5):  acc_u += g ; acc_l += sgn * i s_k g -------------------
template <int MU, int SGN, typename real>
TM_DEV void reconstruct_acc(real *acc, const real *g, real w)
{
    real *au = acc, *al = acc + 12;
    if constexpr (MU == 3) {                    // time: only one half, factor 2 and boundary sign in w
        real *dst = (SGN > 0) ? al : au;
#pragma unroll
        for (int i = 0; i < 12; i++) dst[i] += w * g[i];
    } else {
        const real sw = (real)SGN * w;          // w = 1, or 0 for a hop that leaves a sub-lattice (tm_set_open_dirs)
#pragma unroll
        for (int i = 0; i < 12; i++) au[i] += w * g[i];
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const int a = 2 * c, b = 6 + 2 * c;
            if constexpr (MU == 0) {
                al[a] -= sw * g[b + 1];
                al[a + 1] += sw * g[b];
                al[b] -= sw * g[a + 1];
                al[b + 1] += sw * g[a];
            } else if constexpr (MU == 1) {
                al[a] += sw * g[b];
                al[a + 1] += sw * g[b + 1];
                al[b] -= sw * g[a];
                al[b + 1] -= sw * g[a + 1];
            } else {
                al[a] -= sw * g[a + 1];
                al[a + 1] += sw * g[a];
                al[b] += sw * g[b + 1];
                al[b + 1] -= sw * g[b];
            }
        }
    }
}

// one of the 8 hops.  FWD: U_mu(x) psi(x+mu) with (1 - sgn gamma_mu);  else U_mu(x-mu)^dag psi(x-mu), (1 + sgn gamma_mu).
// a6: the link is fetched (and its third row rebuilt) once and applied to every flavor.
// H = hop number (+x -x +y -y +z -z +t -t).  `lp` = site pointer of the link in global memory, `sp` = site pointer
// of flavor 0 of the neighbour spinor, `lane` = neighbour index & 31.  STG: the link was staged in shared memory
// (tm_stream.cuh) and 7 - H younger cp.async groups may still be pending.
template <typename real> struct TwistIn { real alpha, beta, scale; };      // the twist applied to the INPUT sites (TWIN kernels)
template <int NF, typename real>
TM_DEV void twist(real *w, const real *v, const real *o, real alpha, real beta, real scale);

template <int PREC, int NF, int RECON, int H, bool DAG, bool STG, bool TWIN = false>
TM_DEV void hop(typename PrecTraits<PREC>::real *acc, const char *sp, int lane, const char *lp, int llane,
                typename PrecTraits<PREC>::real w, TwistIn<typename PrecTraits<PREC>::real> ti = TwistIn<typename PrecTraits<PREC>::real>())
{
    typedef typename PrecTraits<PREC>::real real;
    constexpr int MU = H / 2;
    constexpr bool FWD = (H % 2) == 0;
    constexpr int SGN = (FWD != DAG) ? +1 : -1;     // projector sign: forward carries (1 - gamma) unless daggered
    real u[18];
    if constexpr (STG) {
        cp_async_wait<7 - H>();
        load_link<PREC, RECON, true>(u, stage_slot<PREC, RECON>(H), threadIdx.x & 31);
    } else {
        load_link<PREC, RECON, false>(u, lp, llane);
    }
    if constexpr (TWIN) {
        // D R^-1: the neighbour spinor is twisted in registers before the projection.  gamma5 mixes the upper and lower spin
        // halves and tau1 the flavors, so every hop (the time hops too) reads the whole neighbour site, all flavors.
        real v[NF * 24], tv[NF * 24];
#pragma unroll
        for (int f = 0; f < NF; f++) load_spinor<PREC, 0>(v + 24 * f, sp + f * spinor_tile_bytes(PREC), lane);
#pragma unroll
        for (int f = 0; f < NF; f++) twist<NF>(tv + 24 * f, v + 24 * f, v + 24 * (NF - 1 - f), f == 0 ? ti.alpha : -ti.alpha, ti.beta, ti.scale);
#pragma unroll
        for (int f = 0; f < NF; f++) {
            real h[12], g[12];
            if constexpr (MU == 3) {
#pragma unroll
                for (int i = 0; i < 12; i++) h[i] = (SGN > 0) ? tv[24 * f + 12 + i] : tv[24 * f + i];
            } else {
                project<MU, SGN>(h, tv + 24 * f);
            }
            su3_mul<!FWD>(g, u, h);
            reconstruct_acc<MU, SGN>(acc + 24 * f, g, w);
        }
        return;
    }
#pragma unroll
    for (int f = 0; f < NF; f++) {
        real h[12], g[12];
        if constexpr (MU == 3) {
            real v[24];
            load_spinor<PREC, (SGN > 0) ? 2 : 1>(v, sp + f * spinor_tile_bytes(PREC), lane);
#pragma unroll
            for (int i = 0; i < 12; i++) h[i] = (SGN > 0) ? v[12 + i] : v[i];
        } else {
            real v[24];
            load_spinor<PREC, 0>(v, sp + f * spinor_tile_bytes(PREC), lane);
            project<MU, SGN>(h, v);
        }
        su3_mul<!FWD>(g, u, h);
        reconstruct_acc<MU, SGN>(acc + 24 * f, g, w);
    }
}

// ---- local twist (a7):  w = scale * (v + i alpha gamma5 v + beta o),  o = the other flavor's v -----
template <int NF, typename real>
TM_DEV void twist(real *w, const real *v, const real *o, real alpha, real beta, real scale)
{
#pragma unroll
    for (int i = 0; i < 12; i += 2) {
        real ur = v[i] - alpha * v[12 + i + 1], ui = v[i + 1] + alpha * v[12 + i];
        real lr = v[12 + i] - alpha * v[i + 1], li = v[12 + i + 1] + alpha * v[i];
        if constexpr (NF == 2) {
            ur += beta * o[i];
            ui += beta * o[i + 1];
            lr += beta * o[12 + i];
            li += beta * o[12 + i + 1];
        }
        w[i] = scale * ur;
        w[i + 1] = scale * ui;
        w[12 + i] = scale * lr;
        w[12 + i + 1] = scale * li;
    }
}

// The fused epilogue: KT 0 = A, 1 = A-xpay, 2 = B, 3 = REC.  acc (NF x 24) is overwritten with the output.
// Flavor f sees tau3 = +1 (f = 0) or -1 (f = 1) and, through beta tau1, the other flavor's vector.
template <int NF, int KT, typename real>
TM_DEV void epilogue(real *acc, const real *xv, real alpha, real beta, real scale, real kappa, real kappa2)
{
    real v[NF * 24], w[NF * 24];
#pragma unroll
    for (int i = 0; i < NF * 24; i++) v[i] = (KT == 2) ? xv[i] : (KT == 3) ? xv[i] + kappa * acc[i] : acc[i];
#pragma unroll
    for (int f = 0; f < NF; f++) twist<NF>(w + 24 * f, v + 24 * f, v + 24 * (NF - 1 - f), f == 0 ? alpha : -alpha, beta, scale);
#pragma unroll
    for (int i = 0; i < NF * 24; i++) {
        if constexpr (KT == 0 || KT == 3) acc[i] = w[i];
        else if constexpr (KT == 1) acc[i] = xv[i] - kappa2 * w[i];
        else acc[i] = w[i] - kappa2 * acc[i];
    }
}


// resident blocks of 128 threads per SM the register allocation of the fp64 degenerate kernel aims at (measured: profiles/r1_tuning.md;
// with 18-real links two blocks and more registers are 3-5 % faster, with 12-real links three: profiles/r2_tuning.md section 6)
#ifndef TM_MINB_8_1
#define TM_MINB_8_1 3
#endif
template <int PREC, int NF, int RECON, int KT, bool DAG, bool STG, bool TWIN = false>
__global__ void __launch_bounds__(128, (PREC == 8 && NF == 1 && !STG) ? (RECON == 18 ? 2 : TM_MINB_8_1) : (PREC == 8 ? 2 : 1)) tm_dslash_generic(const DslashArgs a)
{
    typedef typename PrecTraits<PREC>::real real;
    tm_pdl_enter();
    const int Vh = a.Vh;
    const int vblock = tm_virtual_block(a, blockIdx.x);
    prefetch_tile<PREC, NF, RECON, KT != 0>(a, blockDim.x, vblock);
    const int site = vblock * blockDim.x + threadIdx.x;        // one thread per output site, all flavors
    if (site >= Vh) return;

    // a2: site decode and neighbours
    const int Xh = a.Xh;
    int r = tm_div(site, a.dXh);
    const int xh = site - r * Xh;
    int r2 = tm_div(r, a.dY);
    const int y = r - r2 * a.Y;
    const int t = tm_div(r2, a.dZ);
    const int z = r2 - t * a.Z;
    const int q = (y + z + t + a.parity) & 1;       // x1 = 2 xh + q
    const int sy = Xh, sz = Xh * a.Y, st = Xh * a.Y * a.Z;
    const int xp = q ? ((xh + 1 == Xh) ? site - (Xh - 1) : site + 1) : site;
    const int xm = q ? site : ((xh == 0) ? site + (Xh - 1) : site - 1);
    const int yp = (y == a.Y - 1) ? site - (a.Y - 1) * sy : site + sy;
    const int ym = (y == 0) ? site + (a.Y - 1) * sy : site - sy;
    const int zp = (z == a.Z - 1) ? site - (a.Z - 1) * sz : site + sz;
    const int zm = (z == 0) ? site + (a.Z - 1) * sz : site - sz;
    const int tp = (t == a.T - 1) ? site - (a.T - 1) * st : site + st;
    const int tm = (t == 0) ? site + (a.T - 1) * st : site - st;
    const real wtp = (real)2 * ((t == a.T - 1) ? (real)a.tbound : (real)1);
    const real wtm = (real)2 * ((t == 0) ? (real)a.tbound : (real)1);
    // y / z hops that wrap: weight 1, or 0 when that direction is cut between GPUs (tm_halo.cu supplies the hop)
    const real wyp = (y == a.Y - 1) ? (real)a.wrap_y : (real)1, wym = (y == 0) ? (real)a.wrap_y : (real)1;
    const real wzp = (z == a.Z - 1) ? (real)a.wrap_z : (real)1, wzm = (z == 0) ? (real)a.wrap_z : (real)1;

    const int nbr[8] = {xp, xm, yp, ym, zp, zm, tp, tm};
    const char *in = static_cast<const char *>(a.in);
    const size_t PB = (size_t)tm_tiles(Vh) * 4 * link_tile_bytes(PREC, RECON);              // one parity's gauge block
    const char *gf = static_cast<const char *>(a.gauge) + (size_t)a.parity * PB;            // U_mu(x)
    const char *gb = static_cast<const char *>(a.gauge) + (size_t)(1 - a.parity) * PB;      // U_mu(x - mu)
    const int lane = site & (TM_TILE - 1);
    const char *lf = gf + link_site_off(PREC, RECON, site, 0);                              // + mu * link_tile_bytes

    // a4 (staged): start all 8 link copies now; hops consume them in order
    if constexpr (STG) {
#pragma unroll
        for (int h = 0; h < 8; h++)
            stage_link<PREC, RECON>(h, (h & 1) ? gb + link_site_off(PREC, RECON, nbr[h], h >> 1) : lf + (h >> 1) * link_tile_bytes(PREC, RECON),
                                    ((h & 1) ? nbr[h] : site) & (TM_TILE - 1));
    }
    real acc[NF * 24];
#pragma unroll
    for (int i = 0; i < NF * 24; i++) acc[i] = 0;

    TwistIn<real> ti;
    ti.alpha = (real)a.alpha_in; ti.beta = (real)a.beta_in; ti.scale = (real)a.scale_in;
#define TM_HOP(H, W)                                                                                              \
    hop<PREC, NF, RECON, (H), DAG, STG, TWIN>(acc, in + spinor_site_off(PREC, NF, nbr[(H)], 0), nbr[(H)] & (TM_TILE - 1),  \
                                        ((H) & 1) ? gb + link_site_off(PREC, RECON, nbr[(H)], (H) >> 1)             \
                                                  : lf + ((H) >> 1) * link_tile_bytes(PREC, RECON),                 \
                                        ((H) & 1) ? (nbr[(H)] & (TM_TILE - 1)) : lane, (W), ti)
    TM_HOP(0, (real)1); TM_HOP(1, (real)1); TM_HOP(2, wyp); TM_HOP(3, wym);
    TM_HOP(4, wzp); TM_HOP(5, wzm); TM_HOP(6, wtp); TM_HOP(7, wtm);
#undef TM_HOP

    // a7: fused local epilogue
    real xv[NF * 24];
    if constexpr (KT != 0) {
        const char *xs = static_cast<const char *>(a.x) + spinor_site_off(PREC, NF, site, 0);
#pragma unroll
        for (int f = 0; f < NF; f++) load_spinor<PREC, 0>(xv + 24 * f, xs + f * spinor_tile_bytes(PREC), lane);
    }
    epilogue<NF, KT>(acc, xv, (real)a.alpha, (real)a.beta, (real)a.scale, (real)a.kappa, (real)a.kappa2);

    // a8: single store
    char *os = static_cast<char *>(a.out) + spinor_site_off(PREC, NF, site, 0);
#pragma unroll
    for (int f = 0; f < NF; f++) store_spinor<PREC>(acc + 24 * f, os + f * spinor_tile_bytes(PREC), lane);
}

template <int PREC, int NF, int RECON, int KT, bool DAG, bool STG, bool TWIN = false>
cudaError_t tm_launch_generic(const DslashArgs &a, cudaStream_t s)
{
    const int threads = a.block_threads;
    const int blocks = (a.Vh + threads - 1) / threads;
    const size_t smem = STG ? (size_t)8 * RECON * PREC * threads : 0;
    if (smem > 48 * 1024) {
        static std::atomic<unsigned long long> raised{0};      // per instantiation, one bit per device
        cudaError_t e = tm_raise_smem(tm_dslash_generic<PREC, NF, RECON, KT, DAG, STG, TWIN>, raised);
        if (e != cudaSuccess) return e;
    }
    return tm_launch_kernel(tm_dslash_generic<PREC, NF, RECON, KT, DAG, STG, TWIN>, a.pdl, blocks, threads, smem, s, a);
}

// table index: [recon 18 / 12 / 8 -> 0 / 1 / 2][kt 0..3][dagger 0..1][staged 0..1]; 8-real links are never staged
#define TM_GENERIC_ROW8(P, N, K)                                                                            \
    {tm_launch_generic<P, N, 8, K, false, false>, "generic<" #P "," #N ",8," #K ",plain>"},                \
    {tm_launch_generic<P, N, 8, K, false, false>, "generic<" #P "," #N ",8," #K ",plain>"},                \
    {tm_launch_generic<P, N, 8, K, true, false>, "generic<" #P "," #N ",8," #K ",dagger>"},                \
    {tm_launch_generic<P, N, 8, K, true, false>, "generic<" #P "," #N ",8," #K ",dagger>"}
#define TM_GENERIC_ROW(P, N, R, K)                                                                          \
    {tm_launch_generic<P, N, R, K, false, false>, "generic<" #P "," #N "," #R "," #K ",plain>"},           \
    {tm_launch_generic<P, N, R, K, false, true>, "generic_staged<" #P "," #N "," #R "," #K ",plain>"},     \
    {tm_launch_generic<P, N, R, K, true, false>, "generic<" #P "," #N "," #R "," #K ",dagger>"},           \
    {tm_launch_generic<P, N, R, K, true, true>, "generic_staged<" #P "," #N "," #R "," #K ",dagger>"}
// input-twist (D R^-1) kernels, direct loads only: index [recon 18 / 12 / 8 -> 0 / 1 / 2][A, REC -> 0, 1][dagger 0..1]
#define TM_GENERIC_TWIN_ROW(P, N, R)                                                                                 \
    {tm_launch_generic<P, N, R, 0, false, false, true>, "generic_twin<" #P "," #N "," #R ",0,plain>"},              \
    {tm_launch_generic<P, N, R, 0, true, false, true>, "generic_twin<" #P "," #N "," #R ",0,dagger>"},              \
    {tm_launch_generic<P, N, R, 3, false, false, true>, "generic_twin<" #P "," #N "," #R ",3,plain>"},              \
    {tm_launch_generic<P, N, R, 3, true, false, true>, "generic_twin<" #P "," #N "," #R ",3,dagger>"}
#define TM_GENERIC_TABLE(P, N)                                                                        \
    static const TmKernelEntry twin_table_##P##_##N[12] = {TM_GENERIC_TWIN_ROW(P, N, 18), TM_GENERIC_TWIN_ROW(P, N, 12),  \
                                                           TM_GENERIC_TWIN_ROW(P, N, 8)};             \
    const TmKernelEntry *tm_generic_twin_table_##P##_##N() { return twin_table_##P##_##N; }          \
    static const TmKernelEntry table_##P##_##N[48] = {                                               \
        TM_GENERIC_ROW(P, N, 18, 0), TM_GENERIC_ROW(P, N, 18, 1), TM_GENERIC_ROW(P, N, 18, 2),       \
        TM_GENERIC_ROW(P, N, 18, 3), TM_GENERIC_ROW(P, N, 12, 0), TM_GENERIC_ROW(P, N, 12, 1),       \
        TM_GENERIC_ROW(P, N, 12, 2), TM_GENERIC_ROW(P, N, 12, 3), TM_GENERIC_ROW8(P, N, 0),          \
        TM_GENERIC_ROW8(P, N, 1), TM_GENERIC_ROW8(P, N, 2), TM_GENERIC_ROW8(P, N, 3)};               \
    const TmKernelEntry *tm_generic_table_##P##_##N() { return table_##P##_##N; }

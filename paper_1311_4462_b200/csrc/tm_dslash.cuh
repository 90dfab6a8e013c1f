// tm_dslash.cuh -- the generic fused twisted-mass dslash kernel (rows a2-a9 of DESIGN.md).
// One thread per output site (both flavors of a doublet); direct 128-bit read-only loads, neighbour reuse through L1/L2.
// Works for every even lattice with extents >= 4; the tiled TMA path (tm_dslash_tma.cuh) takes over on
// conforming lattices.
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
#pragma unroll
        for (int i = 0; i < 12; i++) au[i] += g[i];
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const int a = 2 * c, b = 6 + 2 * c;
            if constexpr (MU == 0) {
                al[a] -= SGN * g[b + 1];
                al[a + 1] += SGN * g[b];
                al[b] -= SGN * g[a + 1];
                al[b + 1] += SGN * g[a];
            } else if constexpr (MU == 1) {
                al[a] += SGN * g[b];
                al[a + 1] += SGN * g[b + 1];
                al[b] -= SGN * g[a];
                al[b + 1] -= SGN * g[a + 1];
            } else {
                al[a] -= SGN * g[a + 1];
                al[a + 1] += SGN * g[a];
                al[b] += SGN * g[b + 1];
                al[b + 1] -= SGN * g[b];
            }
        }
    }
}

// one of the 8 hops.  FWD: U_mu(x) psi(x+mu) with (1 - sgn gamma_mu);  else U_mu(x-mu)^dag psi(x-mu), (1 + sgn gamma_mu).
// a6: the link is fetched (and its third row rebuilt) once and applied to every flavor.
// STG: the link was staged in shared memory (tm_stream.cuh): L addresses the block's [plane][thread] slots and
// WAITN is the number of younger cp.async groups that may still be pending.
template <int PREC, int NF, int RECON, int MU, bool FWD, bool DAG, bool STG, int WAITN>
TM_DEV void hop(typename PrecTraits<PREC>::real *acc, const char *in, const float *in_norm, size_t fl_bytes,
                const LinkSrc L, int Vh, int nbr, typename PrecTraits<PREC>::real w)
{
    typedef typename PrecTraits<PREC>::real real;
    constexpr int SGN = (FWD != DAG) ? +1 : -1;     // projector sign: forward carries (1 - gamma) unless daggered
    real u[18];
    if constexpr (STG) cp_async_wait<WAITN>();
    load_link<PREC, RECON, STG>(u, L.base, L.stride, L.idx);
#pragma unroll
    for (int f = 0; f < NF; f++) {
        real h[12], g[12];
        if constexpr (MU == 3) {
            real v[24];
            load_spinor<PREC, (SGN > 0) ? 2 : 1>(v, in + f * fl_bytes, in_norm + (size_t)f * Vh, Vh, nbr);
#pragma unroll
            for (int i = 0; i < 12; i++) h[i] = (SGN > 0) ? v[12 + i] : v[i];
        } else {
            real v[24];
            load_spinor<PREC, 0>(v, in + f * fl_bytes, in_norm + (size_t)f * Vh, Vh, nbr);
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


template <int PREC, int NF, int RECON, int KT, bool DAG, bool STG>
__global__ void __launch_bounds__(128, (PREC == 8 && NF == 1 && !STG) ? 3 : (PREC == 8 ? 2 : 1)) tm_dslash_generic(const DslashArgs a)
{
    typedef typename PrecTraits<PREC>::real real;
    constexpr int NCH = PrecTraits<PREC>::NCH;
    const int Vh = a.Vh;
    prefetch_tile<PREC, NF, RECON, KT != 0>(a, blockDim.x, blockIdx.x);
    const int site = blockIdx.x * blockDim.x + threadIdx.x;        // one thread per output site, all flavors
    if (site >= Vh) return;

    // a2: site decode and neighbours
    const int Xh = a.Xh;
    const int xh = site % Xh;
    int r = site / Xh;
    const int y = r % a.Y;
    r /= a.Y;
    const int z = r % a.Z;
    const int t = r / a.Z;
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

    const size_t fl_bytes = (size_t)NCH * Vh * 16;                      // one flavor's chunk block
    const char *in = static_cast<const char *>(a.in);
    const float *in_norm = reinterpret_cast<const float *>(in + NF * fl_bytes);
    const size_t blk = (size_t)RECON * PREC * Vh;                       // one [parity][mu] block
    const char *gf = static_cast<const char *>(a.gauge) + (size_t)a.parity * 4 * blk;        // U_mu(x)
    const char *gb = static_cast<const char *>(a.gauge) + (size_t)(1 - a.parity) * 4 * blk;  // U_mu(x - mu)

    // a4 (staged): start all 8 link copies now; hops consume them in order
    const int nt = blockDim.x, tid = threadIdx.x;
    constexpr int LB = RECON * PREC;                                    // bytes of one stored link
    if constexpr (STG) {
        stage_link<PREC, RECON>(tm_smem + 0 * LB * nt, gf + 0 * blk, Vh, site, nt, tid);
        stage_link<PREC, RECON>(tm_smem + 1 * LB * nt, gb + 0 * blk, Vh, xm, nt, tid);
        stage_link<PREC, RECON>(tm_smem + 2 * LB * nt, gf + 1 * blk, Vh, site, nt, tid);
        stage_link<PREC, RECON>(tm_smem + 3 * LB * nt, gb + 1 * blk, Vh, ym, nt, tid);
        stage_link<PREC, RECON>(tm_smem + 4 * LB * nt, gf + 2 * blk, Vh, site, nt, tid);
        stage_link<PREC, RECON>(tm_smem + 5 * LB * nt, gb + 2 * blk, Vh, zm, nt, tid);
        stage_link<PREC, RECON>(tm_smem + 6 * LB * nt, gf + 3 * blk, Vh, site, nt, tid);
        stage_link<PREC, RECON>(tm_smem + 7 * LB * nt, gb + 3 * blk, Vh, tm, nt, tid);
    }
    real acc[NF * 24];
#pragma unroll
    for (int i = 0; i < NF * 24; i++) acc[i] = 0;

    hop<PREC, NF, RECON, 0, true, DAG, STG, 7>(acc, in, in_norm, fl_bytes, link_src<STG>(0, LB, gf + 0 * blk, Vh, site), Vh, xp, (real)1);
    hop<PREC, NF, RECON, 0, false, DAG, STG, 6>(acc, in, in_norm, fl_bytes, link_src<STG>(1, LB, gb + 0 * blk, Vh, xm), Vh, xm, (real)1);
    hop<PREC, NF, RECON, 1, true, DAG, STG, 5>(acc, in, in_norm, fl_bytes, link_src<STG>(2, LB, gf + 1 * blk, Vh, site), Vh, yp, (real)1);
    hop<PREC, NF, RECON, 1, false, DAG, STG, 4>(acc, in, in_norm, fl_bytes, link_src<STG>(3, LB, gb + 1 * blk, Vh, ym), Vh, ym, (real)1);
    hop<PREC, NF, RECON, 2, true, DAG, STG, 3>(acc, in, in_norm, fl_bytes, link_src<STG>(4, LB, gf + 2 * blk, Vh, site), Vh, zp, (real)1);
    hop<PREC, NF, RECON, 2, false, DAG, STG, 2>(acc, in, in_norm, fl_bytes, link_src<STG>(5, LB, gb + 2 * blk, Vh, zm), Vh, zm, (real)1);
    hop<PREC, NF, RECON, 3, true, DAG, STG, 1>(acc, in, in_norm, fl_bytes, link_src<STG>(6, LB, gf + 3 * blk, Vh, site), Vh, tp, wtp);
    hop<PREC, NF, RECON, 3, false, DAG, STG, 0>(acc, in, in_norm, fl_bytes, link_src<STG>(7, LB, gb + 3 * blk, Vh, tm), Vh, tm, wtm);

    // a7: fused local epilogue
    real xv[NF * 24];
    if constexpr (KT != 0) {
        const char *xb = static_cast<const char *>(a.x);
        const float *xn = reinterpret_cast<const float *>(xb + NF * fl_bytes);
#pragma unroll
        for (int f = 0; f < NF; f++) load_spinor<PREC, 0>(xv + 24 * f, xb + f * fl_bytes, xn + (size_t)f * Vh, Vh, site);
    }
    epilogue<NF, KT>(acc, xv, (real)a.alpha, (real)a.beta, (real)a.scale, (real)a.kappa, (real)a.kappa2);

    // a8: single store
    char *ob = static_cast<char *>(a.out);
    float *on = reinterpret_cast<float *>(ob + NF * fl_bytes);
#pragma unroll
    for (int f = 0; f < NF; f++) store_spinor<PREC>(acc + 24 * f, ob + f * fl_bytes, on + (size_t)f * Vh, Vh, site);
}

template <int PREC, int NF, int RECON, int KT, bool DAG, bool STG>
cudaError_t tm_launch_generic(const DslashArgs &a, cudaStream_t s)
{
    const int threads = a.block_threads;
    const int blocks = (a.Vh + threads - 1) / threads;
    const size_t smem = STG ? (size_t)8 * RECON * PREC * threads : 0;
    if (smem > 48 * 1024) {
        static bool raised = false;      // per instantiation
        if (!raised) {
            cudaError_t e = cudaFuncSetAttribute(tm_dslash_generic<PREC, NF, RECON, KT, DAG, STG>,
                                                 cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
            if (e != cudaSuccess) return e;
            raised = true;
        }
    }
    tm_dslash_generic<PREC, NF, RECON, KT, DAG, STG><<<blocks, threads, smem, s>>>(a);
    return cudaGetLastError();
}

// table index: [recon18?0:1][kt 0..3][dagger 0..1][staged 0..1]
#define TM_GENERIC_ROW(P, N, R, K)                                                                          \
    {tm_launch_generic<P, N, R, K, false, false>, "generic<" #P "," #N "," #R "," #K ",plain>"},           \
    {tm_launch_generic<P, N, R, K, false, true>, "generic_staged<" #P "," #N "," #R "," #K ",plain>"},     \
    {tm_launch_generic<P, N, R, K, true, false>, "generic<" #P "," #N "," #R "," #K ",dagger>"},           \
    {tm_launch_generic<P, N, R, K, true, true>, "generic_staged<" #P "," #N "," #R "," #K ",dagger>"}
#define TM_GENERIC_TABLE(P, N)                                                                        \
    static const TmKernelEntry table_##P##_##N[32] = {                                               \
        TM_GENERIC_ROW(P, N, 18, 0), TM_GENERIC_ROW(P, N, 18, 1), TM_GENERIC_ROW(P, N, 18, 2),       \
        TM_GENERIC_ROW(P, N, 18, 3), TM_GENERIC_ROW(P, N, 12, 0), TM_GENERIC_ROW(P, N, 12, 1),       \
        TM_GENERIC_ROW(P, N, 12, 2), TM_GENERIC_ROW(P, N, 12, 3)};                                   \
    const TmKernelEntry *tm_generic_table_##P##_##N() { return table_##P##_##N; }

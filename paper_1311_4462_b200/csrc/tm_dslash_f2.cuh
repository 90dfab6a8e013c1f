// tm_dslash_f2.cuh -- the fused twisted-mass dslash for fp32 and half, written in packed FP32 (FFMA2, tm_f2.cuh).
// Same operator, boundary handling and thread mapping as the scalar kernel in tm_dslash.cuh (rows a2-a9 of
// DESIGN.md); what changes is the arithmetic: every register pair carries the two spin components
// of one half of the spinor, so projection, SU(3) multiply, reconstruction and twist each take half the issue slots.
//
// Register layout of a spinor S[12]:  S[(half*3 + color)*2 + reim] = (spin 2*half, spin 2*half+1).
// Half-spinor H[6] / G[6]:            H[color*2 + reim]            = (first spin, second spin).
// With sgn = +1 for (1 - gamma_mu), -1 for (1 + gamma_mu), U = upper pairs, L = lower pairs (basis C5):
//   mu=x:  Hr = Ur + sgn sw(Li)          Hi = Ui - sgn sw(Lr)            sw = swap the two lanes
//   mu=y:  Hr = Ur + (-sgn,+sgn) sw(Lr)  Hi = Ui + (-sgn,+sgn) sw(Li)
//   mu=z:  Hr = Ur + (+sgn,-sgn) Li      Hi = Ui + (-sgn,+sgn) Lr
//   mu=t:  H = L (sgn > 0) or U (sgn < 0), weight 2
// and the lower half of the result is  sgn * i sigma_k G  (see reconstruct_f2).
//
// Half precision: int16 are converted with PRMT + one FADD2 per pair (no I2F), the per-site norm and the 1/32767
// of the links are folded into the accumulate weight, and the output is quantised with one FFMA2 + PRMT per pair.
#pragma once
#include "tm_f2.cuh"
#include "tm_internal.h"
#include "tm_layout.cuh"
#include "tm_stream.cuh"

#define TM_INV15 (1.0f / 32767.0f)

// ---- loads ------------------------------------------------------------------------------------------
// PART: 0 all, 1 upper only (S[0..5]), 2 lower only (S[6..11]).  fp32: values; half: RAW integers (scale deferred).
template <int PREC, int PART>
TM_DEV void load_spinor_f2(f2 *S, const char *base, int Vh, int idx)
{
    if constexpr (PREC == 4) {
        constexpr int lo = (PART == 2) ? 3 : 0, hi = (PART == 1) ? 3 : 6;
        const float4 *p = reinterpret_cast<const float4 *>(base) + idx;
#pragma unroll
        for (int k = lo; k < hi; k++) {
            const float4 c = __ldg(p + (size_t)k * Vh);
            S[2 * k] = mk2(c.x, c.y);
            S[2 * k + 1] = mk2(c.z, c.w);
        }
    } else {
        const int4 *p = reinterpret_cast<const int4 *>(base) + idx;
        if constexpr (PART != 2) {
            const int4 c = __ldg(p);
            S[0] = cvt_pair(c.x); S[1] = cvt_pair(c.y); S[2] = cvt_pair(c.z); S[3] = cvt_pair(c.w);
        }
        {
            const int4 c = __ldg(p + (size_t)Vh);
            if constexpr (PART != 2) { S[4] = cvt_pair(c.x); S[5] = cvt_pair(c.y); }
            if constexpr (PART != 1) { S[6] = cvt_pair(c.z); S[7] = cvt_pair(c.w); }
        }
        if constexpr (PART != 1) {
            const int4 c = __ldg(p + (size_t)2 * Vh);
            S[8] = cvt_pair(c.x); S[9] = cvt_pair(c.y); S[10] = cvt_pair(c.z); S[11] = cvt_pair(c.w);
        }
    }
}

// Link as 9 (re, im) pairs W[row*3+col]; half: RAW integers for rows 0,1 (12-real: row 2 rebuilt and rescaled to
// the same raw scale).  a4 of DESIGN.md.
template <int PREC, int RECON, bool SM>
TM_DEV void load_link_f2(f2 *W, const char *base, int Vh, int idx)
{
    if constexpr (PREC == 4) {
        constexpr int NF4 = (RECON == 18) ? 4 : 3;
#pragma unroll
        for (int k = 0; k < NF4; k++) {
            const float4 c = ld_f4<SM>(base + ((size_t)k * Vh + idx) * 16);
            W[2 * k] = mk2(c.x, c.y);
            W[2 * k + 1] = mk2(c.z, c.w);
        }
        if constexpr (RECON == 18) {
            const float2 c = ld_f2<SM>(base + (size_t)4 * Vh * 16 + (size_t)idx * 8);
            W[8] = mk2(c.x, c.y);
        }
    } else {
        const int4 c = ld_i4<SM>(base + (size_t)idx * 16);
        W[0] = cvt_pair(c.x); W[1] = cvt_pair(c.y); W[2] = cvt_pair(c.z); W[3] = cvt_pair(c.w);
        if constexpr (RECON == 18) {
            const int4 d = ld_i4<SM>(base + ((size_t)Vh + idx) * 16);
            W[4] = cvt_pair(d.x); W[5] = cvt_pair(d.y); W[6] = cvt_pair(d.z); W[7] = cvt_pair(d.w);
            W[8] = cvt_pair(ld_i1<SM>(base + (size_t)2 * Vh * 16 + (size_t)idx * 4));
        } else {
            const int2 d = ld_i2<SM>(base + (size_t)Vh * 16 + (size_t)idx * 8);
            W[4] = cvt_pair(d.x); W[5] = cvt_pair(d.y);
        }
    }
    if constexpr (RECON == 12) {
        // row2[c] = conj(row0[c1] row1[c2] - row0[c2] row1[c1]),  pairs are (re, im):
        //   S = a.re*b - c.re*d ,  T = a.im*sw(b) - c.im*sw(d) ;  a*b - c*d = (S.x - T.x, S.y + T.y)
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
            const f2 A = W[c1], B = W[3 + c2], C = W[c2], D = W[3 + c1];
            const f2 S = fma2(bc2(-C.x), D, mul2(bc2(A.x), B));
            const f2 T = fma2(bc2(-C.y), sw2(D), mul2(bc2(A.y), sw2(B)));
            float re = S.x - T.x, im = -S.y - T.y;
            if constexpr (PREC == 2) { re *= TM_INV15; im *= TM_INV15; }     // raw * raw / 32767 -> raw scale
            W[6 + c] = mk2(re, im);
        }
    }
}

// ---- a3: spin projection, packed ----------------------------------------------------------------------
template <int MU, int SGN>
TM_DEV void project_f2(f2 *H, const f2 *S)
{
    const f2 *U = S, *L = S + 6;
    const f2 pm = mk2((float)SGN, (float)-SGN), mp = mk2((float)-SGN, (float)SGN);
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const f2 Ur = U[2 * c], Ui = U[2 * c + 1], Lr = L[2 * c], Li = L[2 * c + 1];
        if constexpr (MU == 0) {
            H[2 * c] = fma2(sw2(Li), bc2((float)SGN), Ur);
            H[2 * c + 1] = fma2(sw2(Lr), bc2((float)-SGN), Ui);
        } else if constexpr (MU == 1) {
            H[2 * c] = fma2(sw2(Lr), mp, Ur);
            H[2 * c + 1] = fma2(sw2(Li), mp, Ui);
        } else {
            H[2 * c] = fma2(Li, pm, Ur);
            H[2 * c + 1] = fma2(Lr, mp, Ui);
        }
    }
}

// ---- a5: color multiply on both spin components at once: 36 packed instructions ------------------------
template <bool ADJ>
TM_DEV void su3_mul_f2(f2 *G, const f2 *W, const f2 *H)
{
#pragma unroll
    for (int c = 0; c < 3; c++) {
        f2 re, im;
#pragma unroll
        for (int d = 0; d < 3; d++) {
            const f2 w = ADJ ? W[3 * d + c] : W[3 * c + d];
            const float ur = w.x, ui = ADJ ? -w.y : w.y;
            if (d == 0) {
                re = mul2(bc2(ur), H[2 * d]);
                im = mul2(bc2(ur), H[2 * d + 1]);
            } else {
                re = fma2(bc2(ur), H[2 * d], re);
                im = fma2(bc2(ur), H[2 * d + 1], im);
            }
            re = fma2(bc2(-ui), H[2 * d + 1], re);
            im = fma2(bc2(ui), H[2 * d], im);
        }
        G[2 * c] = re;
        G[2 * c + 1] = im;
    }
}

// ---- a5: reconstruction + accumulate with weight w:  A_u += w G ;  A_l += w sgn i sigma_k G -----------
//   x: (i s1 g) = (i g1, i g0)  -> Alr += -sgn sw(Gi), Ali += +sgn sw(Gr)
//   y: (i s2 g) = (g1, -g0)     -> Alr += (sgn,-sgn) sw(Gr), Ali += (sgn,-sgn) sw(Gi)
//   z: (i s3 g) = (i g0, -i g1) -> Alr += (-sgn,sgn) Gi,     Ali += (sgn,-sgn) Gr
template <int MU, int SGN>
TM_DEV void reconstruct_f2(f2 *A, const f2 *G, float w)
{
    f2 *Au = A, *Al = A + 6;
    if constexpr (MU == 3) {
        f2 *dst = (SGN > 0) ? Al : Au;
#pragma unroll
        for (int i = 0; i < 6; i++) dst[i] = fma2(G[i], bc2(w), dst[i]);
    } else {
        const float sw_ = (float)SGN * w;
        const f2 pm = mk2(sw_, -sw_), mp = mk2(-sw_, sw_);
#pragma unroll
        for (int i = 0; i < 6; i++) Au[i] = fma2(G[i], bc2(w), Au[i]);
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const f2 Gr = G[2 * c], Gi = G[2 * c + 1];
            if constexpr (MU == 0) {
                Al[2 * c] = fma2(sw2(Gi), bc2(-sw_), Al[2 * c]);
                Al[2 * c + 1] = fma2(sw2(Gr), bc2(sw_), Al[2 * c + 1]);
            } else if constexpr (MU == 1) {
                Al[2 * c] = fma2(sw2(Gr), pm, Al[2 * c]);
                Al[2 * c + 1] = fma2(sw2(Gi), pm, Al[2 * c + 1]);
            } else {
                Al[2 * c] = fma2(Gi, mp, Al[2 * c]);
                Al[2 * c + 1] = fma2(Gr, pm, Al[2 * c + 1]);
            }
        }
    }
}

// a6: the link is fetched, converted and rebuilt once and applied to every flavor.
template <int PREC, int NF, int RECON, int MU, bool FWD, bool DAG, bool STG, int WAITN>
TM_DEV void hop_f2(f2 *A, const char *in, const float *in_norm, size_t fl_bytes, const LinkSrc L, int Vh, int nbr, float w)
{
    constexpr int SGN = (FWD != DAG) ? +1 : -1;
    f2 W[9];
    if constexpr (STG) cp_async_wait<WAITN>();
    load_link_f2<PREC, RECON, STG>(W, L.base, L.stride, L.idx);
#pragma unroll
    for (int f = 0; f < NF; f++) {
        f2 S[12], H[6], G[6];
        const char *inf = in + f * fl_bytes;
        if constexpr (MU == 3) {
            load_spinor_f2<PREC, (SGN > 0) ? 2 : 1>(S, inf, Vh, nbr);
#pragma unroll
            for (int i = 0; i < 6; i++) H[i] = (SGN > 0) ? S[6 + i] : S[i];
        } else {
            load_spinor_f2<PREC, 0>(S, inf, Vh, nbr);
            project_f2<MU, SGN>(H, S);
        }
        float wf = w;
        if constexpr (PREC == 2) wf *= __ldg(in_norm + (size_t)f * Vh + nbr) * (TM_INV15 * TM_INV15);   // site norm x link scale
        su3_mul_f2<!FWD>(G, W, H);
        reconstruct_f2<MU, SGN>(A + 12 * f, G, wf);
    }
}

// ---- a7: local twist, packed:  W = scale (V + i alpha gamma5 V + beta O) ------------------------------
template <int NF>
TM_DEV void twist_f2(f2 *Wo, const f2 *V, const f2 *O, float alpha, float beta, float scale)
{
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int ur = 2 * c, ui = 2 * c + 1, lr = 6 + 2 * c, li = 6 + 2 * c + 1;
        f2 a = fma2(V[li], bc2(-alpha), V[ur]);
        f2 b = fma2(V[lr], bc2(alpha), V[ui]);
        f2 d = fma2(V[ui], bc2(-alpha), V[lr]);
        f2 e = fma2(V[ur], bc2(alpha), V[li]);
        if constexpr (NF == 2) {
            a = fma2(O[ur], bc2(beta), a);
            b = fma2(O[ui], bc2(beta), b);
            d = fma2(O[lr], bc2(beta), d);
            e = fma2(O[li], bc2(beta), e);
        }
        Wo[ur] = mul2(a, bc2(scale));
        Wo[ui] = mul2(b, bc2(scale));
        Wo[lr] = mul2(d, bc2(scale));
        Wo[li] = mul2(e, bc2(scale));
    }
}

// A (NF x 12 pairs) is overwritten with the output; flavor f sees tau3 = +1 (f = 0) / -1 (f = 1) and the other flavor.
template <int NF, int KT>
TM_DEV void epilogue_f2(f2 *A, const f2 *X, float alpha, float beta, float scale, float kappa, float kappa2)
{
    f2 V[NF * 12], Wt[NF * 12];
#pragma unroll
    for (int i = 0; i < NF * 12; i++) V[i] = (KT == 2) ? X[i] : (KT == 3) ? fma2(A[i], bc2(kappa), X[i]) : A[i];
#pragma unroll
    for (int f = 0; f < NF; f++) twist_f2<NF>(Wt + 12 * f, V + 12 * f, V + 12 * (NF - 1 - f), f == 0 ? alpha : -alpha, beta, scale);
#pragma unroll
    for (int i = 0; i < NF * 12; i++) {
        if constexpr (KT == 0 || KT == 3) A[i] = Wt[i];
        else if constexpr (KT == 1) A[i] = fma2(Wt[i], bc2(-kappa2), X[i]);
        else A[i] = fma2(A[i], bc2(-kappa2), Wt[i]);
    }
}

// ---- a8: single store -----------------------------------------------------------------------------------
template <int PREC>
TM_DEV void store_spinor_f2(const f2 *A, char *base, float *norm, int Vh, int idx)
{
    if constexpr (PREC == 4) {
        float4 *p = reinterpret_cast<float4 *>(base) + idx;
#pragma unroll
        for (int k = 0; k < 6; k++) p[(size_t)k * Vh] = make_float4(A[2 * k].x, A[2 * k].y, A[2 * k + 1].x, A[2 * k + 1].y);
    } else {
        float m = 0.f;
#pragma unroll
        for (int i = 0; i < 12; i++) m = fmaxf(m, fmaxf(fabsf(A[i].x), fabsf(A[i].y)));
        const float s = (m > 0.f) ? __fdividef(32767.0f, m) : 0.f;
        int4 *p = reinterpret_cast<int4 *>(base) + idx;
#pragma unroll
        for (int k = 0; k < 3; k++) {
            int4 c;
            c.x = quant_pair(A[4 * k], s);
            c.y = quant_pair(A[4 * k + 1], s);
            c.z = quant_pair(A[4 * k + 2], s);
            c.w = quant_pair(A[4 * k + 3], s);
            p[(size_t)k * Vh] = c;
        }
        norm[idx] = m;
    }
}

template <int PREC, int NF, int RECON, int KT, bool DAG, bool STG>
__global__ void __launch_bounds__(128) tm_dslash_f2(const DslashArgs a)
{
    constexpr int NCH = PrecTraits<PREC>::NCH;
    const int Vh = a.Vh;
    prefetch_tile<PREC, NF, RECON, KT != 0>(a, blockDim.x);
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
    const int q = (y + z + t + a.parity) & 1;
    const int sy = Xh, sz = Xh * a.Y, st = Xh * a.Y * a.Z;
    const int xp = q ? ((xh + 1 == Xh) ? site - (Xh - 1) : site + 1) : site;
    const int xm = q ? site : ((xh == 0) ? site + (Xh - 1) : site - 1);
    const int yp = (y == a.Y - 1) ? site - (a.Y - 1) * sy : site + sy;
    const int ym = (y == 0) ? site + (a.Y - 1) * sy : site - sy;
    const int zp = (z == a.Z - 1) ? site - (a.Z - 1) * sz : site + sz;
    const int zm = (z == 0) ? site + (a.Z - 1) * sz : site - sz;
    const int tp = (t == a.T - 1) ? site - (a.T - 1) * st : site + st;
    const int tm = (t == 0) ? site + (a.T - 1) * st : site - st;
    const float wtp = 2.f * ((t == a.T - 1) ? (float)a.tbound : 1.f);
    const float wtm = 2.f * ((t == 0) ? (float)a.tbound : 1.f);

    const size_t fl_bytes = (size_t)NCH * Vh * 16;
    const char *in = static_cast<const char *>(a.in);
    const float *in_norm = reinterpret_cast<const float *>(in + NF * fl_bytes);
    const size_t blk = (size_t)RECON * PREC * Vh;
    const char *gf = static_cast<const char *>(a.gauge) + (size_t)a.parity * 4 * blk;
    const char *gb = static_cast<const char *>(a.gauge) + (size_t)(1 - a.parity) * 4 * blk;

    const int nt = blockDim.x, tid = threadIdx.x;
    constexpr int LB = RECON * PREC;
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

    f2 A[NF * 12];
#pragma unroll
    for (int i = 0; i < NF * 12; i++) A[i] = mk2(0.f, 0.f);

    hop_f2<PREC, NF, RECON, 0, true, DAG, STG, 7>(A, in, in_norm, fl_bytes, link_src<STG>(0, LB, gf + 0 * blk, Vh, site), Vh, xp, 1.f);
    hop_f2<PREC, NF, RECON, 0, false, DAG, STG, 6>(A, in, in_norm, fl_bytes, link_src<STG>(1, LB, gb + 0 * blk, Vh, xm), Vh, xm, 1.f);
    hop_f2<PREC, NF, RECON, 1, true, DAG, STG, 5>(A, in, in_norm, fl_bytes, link_src<STG>(2, LB, gf + 1 * blk, Vh, site), Vh, yp, 1.f);
    hop_f2<PREC, NF, RECON, 1, false, DAG, STG, 4>(A, in, in_norm, fl_bytes, link_src<STG>(3, LB, gb + 1 * blk, Vh, ym), Vh, ym, 1.f);
    hop_f2<PREC, NF, RECON, 2, true, DAG, STG, 3>(A, in, in_norm, fl_bytes, link_src<STG>(4, LB, gf + 2 * blk, Vh, site), Vh, zp, 1.f);
    hop_f2<PREC, NF, RECON, 2, false, DAG, STG, 2>(A, in, in_norm, fl_bytes, link_src<STG>(5, LB, gb + 2 * blk, Vh, zm), Vh, zm, 1.f);
    hop_f2<PREC, NF, RECON, 3, true, DAG, STG, 1>(A, in, in_norm, fl_bytes, link_src<STG>(6, LB, gf + 3 * blk, Vh, site), Vh, tp, wtp);
    hop_f2<PREC, NF, RECON, 3, false, DAG, STG, 0>(A, in, in_norm, fl_bytes, link_src<STG>(7, LB, gb + 3 * blk, Vh, tm), Vh, tm, wtm);

    f2 X[NF * 12];
    if constexpr (KT != 0) {
        const char *xb = static_cast<const char *>(a.x);
        const float *xn = reinterpret_cast<const float *>(xb + NF * fl_bytes);
#pragma unroll
        for (int f = 0; f < NF; f++) {
            load_spinor_f2<PREC, 0>(X + 12 * f, xb + f * fl_bytes, Vh, site);
            if constexpr (PREC == 2) {
                const float s = __ldg(xn + (size_t)f * Vh + site) * TM_INV15;
#pragma unroll
                for (int i = 0; i < 12; i++) X[12 * f + i] = mul2(X[12 * f + i], bc2(s));
            }
        }
    }
    epilogue_f2<NF, KT>(A, X, (float)a.alpha, (float)a.beta, (float)a.scale, (float)a.kappa, (float)a.kappa2);

    char *ob = static_cast<char *>(a.out);
    float *on = reinterpret_cast<float *>(ob + NF * fl_bytes);
#pragma unroll
    for (int f = 0; f < NF; f++) store_spinor_f2<PREC>(A + 12 * f, ob + f * fl_bytes, on + (size_t)f * Vh, Vh, site);
}

template <int PREC, int NF, int RECON, int KT, bool DAG, bool STG>
cudaError_t tm_launch_f2(const DslashArgs &a, cudaStream_t s)
{
    const int threads = a.block_threads;
    const int blocks = (a.Vh + threads - 1) / threads;
    const size_t smem = STG ? (size_t)8 * RECON * PREC * threads : 0;
    if (smem > 48 * 1024) {
        static bool raised = false;      // per instantiation
        if (!raised) {
            cudaError_t e = cudaFuncSetAttribute(tm_dslash_f2<PREC, NF, RECON, KT, DAG, STG>,
                                                 cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
            if (e != cudaSuccess) return e;
            raised = true;
        }
    }
    tm_dslash_f2<PREC, NF, RECON, KT, DAG, STG><<<blocks, threads, smem, s>>>(a);
    return cudaGetLastError();
}

// table index: [recon18?0:1][kt 0..3][dagger 0..1][staged 0..1]
#define TM_F2_ROW(P, N, R, K)                                                                       \
    {tm_launch_f2<P, N, R, K, false, false>, "f2<" #P "," #N "," #R "," #K ",plain>"},             \
    {tm_launch_f2<P, N, R, K, false, true>, "f2_staged<" #P "," #N "," #R "," #K ",plain>"},       \
    {tm_launch_f2<P, N, R, K, true, false>, "f2<" #P "," #N "," #R "," #K ",dagger>"},             \
    {tm_launch_f2<P, N, R, K, true, true>, "f2_staged<" #P "," #N "," #R "," #K ",dagger>"}
#define TM_F2_TABLE(P, N)                                                                    \
    static const TmKernelEntry f2table_##P##_##N[32] = {                                    \
        TM_F2_ROW(P, N, 18, 0), TM_F2_ROW(P, N, 18, 1), TM_F2_ROW(P, N, 18, 2),             \
        TM_F2_ROW(P, N, 18, 3), TM_F2_ROW(P, N, 12, 0), TM_F2_ROW(P, N, 12, 1),             \
        TM_F2_ROW(P, N, 12, 2), TM_F2_ROW(P, N, 12, 3)};                                    \
    const TmKernelEntry *tm_f2_table_##P##_##N() { return f2table_##P##_##N; }

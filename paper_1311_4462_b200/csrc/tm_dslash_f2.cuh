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

// Software-pipeline depth (hops of loads in flight ahead of the arithmetic) per (precision, flavors); chosen by
// measurement on B200 (profiles/), overridable at compile time for sweeps.
#ifndef TM_PD_4_1
#define TM_PD_4_1 1
#endif
#ifndef TM_PD_4_2
#define TM_PD_4_2 1
#endif
#ifndef TM_PD_2_1
#define TM_PD_2_1 0
#endif
#ifndef TM_PD_2_2
#define TM_PD_2_2 1
#endif
// Resident blocks of 128 threads per SM the register allocation aims at (second __launch_bounds__ argument).  It is
// what makes ptxas keep the pipelined loads early: without it the loads are sunk back next to their first use.
#ifndef TM_MINB_4_1
#define TM_MINB_4_1 4
#endif
#ifndef TM_MINB_4_2
#define TM_MINB_4_2 3
#endif
#ifndef TM_MINB_2_1
#define TM_MINB_2_1 3
#endif
#ifndef TM_MINB_2_2
#define TM_MINB_2_2 4
#endif
template <int PREC, int NF> __host__ __device__ constexpr int f2_min_blocks()
{
    return PREC == 4 ? (NF == 1 ? TM_MINB_4_1 : TM_MINB_4_2) : (NF == 1 ? TM_MINB_2_1 : TM_MINB_2_2);
}
template <int PREC, int NF> __host__ __device__ constexpr int f2_pipeline_depth()
{
    return PREC == 4 ? (NF == 1 ? TM_PD_4_1 : TM_PD_4_2) : (NF == 1 ? TM_PD_2_1 : TM_PD_2_2);
}

// ---- loads: issue and use are separate (software pipelining) ------------------------------
// The raw 128-bit words of one hop (link + the neighbour spinor of every flavor + norms) are loaded into a HopRaw
// by issue_*; the arithmetic of that hop reads them PD hops later (consume_hop), so PD + 1 hops of loads are in
// flight per thread while the previous hops are being computed.  Nothing is converted at issue time: in half a hop
// in flight costs 19 registers per flavor-site, in fp32 36 + 24 NF.
template <int PREC, int NF, int RECON>
struct HopRaw {
    static constexpr int NL = (PREC == 4) ? (RECON == 18 ? 4 : RECON == 12 ? 3 : 2) : (RECON == 18 ? 2 : 1);   // 128-bit link words (half 8-real: 1)
    static constexpr int NS = (PREC == 4) ? 6 : 3;                                          // 128-bit spinor words
    uint4 l[NL];
    uint2 lt;            // link tail: fp32/18 float2, half/12 int2, half/18 int (.x)
    uint4 s[NF][NS];
    float n[NF];         // half: site norms
};

// Global loads are volatile asm so that the compiler keeps them where the pipeline puts them (it otherwise sinks
// them back next to their first use to save registers, which serialises load latency and arithmetic hop by hop).
TM_DEV uint4 ldg_nc_u4(const void *p)
{
    uint4 v;
    asm volatile("ld.global.nc.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}
TM_DEV uint2 ldg_nc_u2(const void *p)
{
    uint2 v;
    asm volatile("ld.global.nc.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
    return v;
}
TM_DEV unsigned ldg_nc_u1(const void *p)
{
    unsigned v;
    asm volatile("ld.global.nc.u32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
// link words: from the staged shared-memory copy (SM) or streaming from global memory (L2 evict-first, tm_layout.cuh)
template <bool SM> TM_DEV uint4 ld_u4(const void *p) { if constexpr (SM) return *reinterpret_cast<const uint4 *>(p); else return ldg_stream_u4(p); }
template <bool SM> TM_DEV uint2 ld_u2(const void *p) { if constexpr (SM) return *reinterpret_cast<const uint2 *>(p); else return ldg_stream_u2(p); }
template <bool SM> TM_DEV unsigned ld_u1(const void *p) { if constexpr (SM) return *reinterpret_cast<const unsigned *>(p); else return ldg_stream_u1(p); }

// a4 (fetch): the stored words of one link; `lp` = the link's site pointer in global memory or in the staged copy
template <int PREC, int NF, int RECON, bool SM>
TM_DEV void issue_link(HopRaw<PREC, NF, RECON> &r, const char *lp, int lane)
{
    constexpr int N16 = link_n16<PREC, RECON>();
#pragma unroll
    for (int k = 0; k < N16; k++) r.l[k] = ld_u4<SM>(lp + k * TM_PLANE);
    if constexpr (PREC == 4 && RECON == 18) r.lt = ld_u2<SM>(lp + tail_off(4, 8, lane));
    if constexpr (PREC == 2 && RECON == 18) r.lt.x = ld_u1<SM>(lp + tail_off(2, 4, lane));
    if constexpr (PREC == 2 && RECON == 12) r.lt = ld_u2<SM>(lp + tail_off(1, 8, lane));
}

// PART: 0 all, 1 upper half only, 2 lower half only (time hops, a3).  `sp` = site pointer of flavor 0.
template <int PREC, int NF, int RECON, int PART>
TM_DEV void issue_spinor(HopRaw<PREC, NF, RECON> &r, const char *sp, int lane)
{
#pragma unroll
    for (int f = 0; f < NF; f++) {
        const char *p = sp + f * spinor_tile_bytes(PREC);
        if constexpr (PREC == 4) {
            constexpr int lo = (PART == 2) ? 3 : 0, hi = (PART == 1) ? 3 : 6;
#pragma unroll
            for (int k = lo; k < hi; k++) r.s[f][k] = ldg_nc_u4(p + k * TM_PLANE);
        } else {
            if constexpr (PART != 2) r.s[f][0] = ldg_nc_u4(p);
            r.s[f][1] = ldg_nc_u4(p + TM_PLANE);
            if constexpr (PART != 1) r.s[f][2] = ldg_nc_u4(p + 2 * TM_PLANE);
            r.n[f] = __uint_as_float(ldg_nc_u1(p + tail_off(3, 4, lane)));
        }
    }
}

// raw words -> pairs.  fp32: values; half: RAW integers as floats (scale deferred), or BIASED: raw + TM_CVT_MAGIC
// (the bias is removed for free by the projection).  Only the PART's pairs are valid.
template <int PREC, int PART, bool BIASED = false>
TM_DEV void raw_to_spinor(f2 *S, const uint4 *s)
{
    if constexpr (PREC == 4) {
        constexpr int lo = (PART == 2) ? 3 : 0, hi = (PART == 1) ? 3 : 6;
#pragma unroll
        for (int k = lo; k < hi; k++) {
            S[2 * k] = mk2(__uint_as_float(s[k].x), __uint_as_float(s[k].y));
            S[2 * k + 1] = mk2(__uint_as_float(s[k].z), __uint_as_float(s[k].w));
        }
    } else {
        auto cv = [](uint32_t w) { if constexpr (BIASED) return cvt_pair_biased(w); else return cvt_pair(w); };
        if constexpr (PART != 2) {
            S[0] = cv(s[0].x); S[1] = cv(s[0].y); S[2] = cv(s[0].z); S[3] = cv(s[0].w);
            S[4] = cv(s[1].x); S[5] = cv(s[1].y);
        }
        if constexpr (PART != 1) {
            S[6] = cv(s[1].z); S[7] = cv(s[1].w);
            S[8] = cv(s[2].x); S[9] = cv(s[2].y); S[10] = cv(s[2].z); S[11] = cv(s[2].w);
        }
    }
}

// a4 (rebuild): link as 9 (re, im) pairs W[row*3+col]; half: RAW integers for rows 0,1; 12-real: row 2 is rebuilt and,
// in half, left at raw x raw scale: the factor 1/32767 is applied where it is cheapest (consume_hop).
// 8-real links, fp32 (chart: tm_layout.cuh rebuild_from8): rows 0 and 1 from the 8 stored reals with the fast
// special-function unit (sin / cos / rsqrt / rcp approximations, abs. error ~5e-7: inside the fp32 tolerance; the
// scalar kernels use the IEEE forms).  Scalar arithmetic: the link is per site, not per spin pair.
TM_DEV void rows01_from8_fast(f2 *W, const float *p)
{
    const float a2r = p[0], a2i = p[1], a3r = p[2], a3i = p[3], b1r = p[4], b1i = p[5];
    const float N = fmaf(a2r, a2r, fmaf(a2i, a2i, fmaf(a3r, a3r, a3i * a3i)));
#ifndef TM_RECON8_ACCURATE      /* IEEE sincospi / division: 20-30 % slower (profiles/r2_tuning.md), no faster than 12-real links */
    const float t1 = p[6] * 3.14159265358979f, t2 = p[7] * 3.14159265358979f;
    const float s1 = __sinf(t1), c1 = __cosf(t1), s2 = __sinf(t2), c2 = __cosf(t2);
#else
    float s1, c1, s2, c2;
    sincospif(p[6], &s1, &c1);
    sincospif(p[7], &s2, &c2);
#endif
    const float q1 = fmaxf(1.f - N, 0.f), q2 = fmaxf(N - fmaf(b1r, b1r, b1i * b1i), 0.f);
    const float m1 = q1 * rsqrtf(fmaxf(q1, 1e-30f)), m2 = q2 * rsqrtf(fmaxf(q2, 1e-30f));
    const float a1r = m1 * c1, a1i = m1 * s1;
    const float r2r = m2 * c2, r2i = -(m2 * s2);                                        // conj(c1)
    const float r1r = -fmaf(a1r, b1r, a1i * b1i), r1i = fmaf(a1i, b1r, -(a1r * b1i));   // -conj(a1) b1
#ifndef TM_RECON8_ACCURATE      /* IEEE sincospi / division: 20-30 % slower (profiles/r2_tuning.md), no faster than 12-real links */
    const float iN = __fdividef(1.f, N);
#else
    const float iN = 1.f / N;
#endif
    W[0] = mk2(a1r, a1i);
    W[1] = mk2(a2r, a2i);
    W[2] = mk2(a3r, a3i);
    W[3] = mk2(b1r, b1i);
    W[4] = mk2((fmaf(r1r, a2r, -(r1i * a2i)) - fmaf(a3r, r2r, a3i * r2i)) * iN,
               (fmaf(r1r, a2i, r1i * a2r) - fmaf(a3r, r2i, -(a3i * r2r))) * iN);
    W[5] = mk2((fmaf(a2r, r2r, a2i * r2i) + fmaf(a3r, r1r, -(a3i * r1i))) * iN,
               (fmaf(a2r, r2i, -(a2i * r2r)) + fmaf(a3r, r1i, a3i * r1r)) * iN);
}

// row2[c] = conj(row0[c1] row1[c2] - row0[c2] row1[c1]),  pairs are (re, im):
//   S = a.re*b - c.re*d ,  T = a.im*sw(b) - c.im*sw(d) ;  a*b - c*d = (S.x - T.x, S.y + T.y)
// half: row 2 stays at raw * raw scale (32767 x the raw scale of rows 0, 1); consume_hop compensates
TM_DEV void link_row2_f2(f2 *W)
{
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
        const f2 A = W[c1], B = W[3 + c2], C = W[c2], D = W[3 + c1];
        const f2 S = fma2(bc2(-C.x), D, mul2(bc2(A.x), B));
        const f2 T = fma2(bc2(-C.y), sw2(D), mul2(bc2(A.y), sw2(B)));
        W[6 + c] = mk2(S.x - T.x, -S.y - T.y);
    }
}

template <int PREC, int NF, int RECON>
TM_DEV void raw_to_link(f2 *W, const HopRaw<PREC, NF, RECON> &r)
{
    if constexpr (RECON == 8 && PREC == 4) {
        const float p[8] = {__uint_as_float(r.l[0].x), __uint_as_float(r.l[0].y), __uint_as_float(r.l[0].z), __uint_as_float(r.l[0].w),
                            __uint_as_float(r.l[1].x), __uint_as_float(r.l[1].y), __uint_as_float(r.l[1].z), __uint_as_float(r.l[1].w)};
        rows01_from8_fast(W, p);
    } else if constexpr (RECON == 8) {
        // half: the 8 stored reals are one 128-bit word of int16 at scale 32767; the rebuilt rows come out at TRUE scale
        // (consume_hop then folds only the spinor's 1 / 32767 into the weight)
        const f2 a = mul2(cvt_pair(r.l[0].x), bc2(TM_INV15)), b = mul2(cvt_pair(r.l[0].y), bc2(TM_INV15));
        const f2 c = mul2(cvt_pair(r.l[0].z), bc2(TM_INV15)), d = mul2(cvt_pair(r.l[0].w), bc2(TM_INV15));
        const float p[8] = {a.x, a.y, b.x, b.y, c.x, c.y, d.x, d.y};
        rows01_from8_fast(W, p);
    } else if constexpr (PREC == 4) {
#pragma unroll
        for (int k = 0; k < HopRaw<PREC, NF, RECON>::NL; k++) {
            W[2 * k] = mk2(__uint_as_float(r.l[k].x), __uint_as_float(r.l[k].y));
            W[2 * k + 1] = mk2(__uint_as_float(r.l[k].z), __uint_as_float(r.l[k].w));
        }
        if constexpr (RECON == 18) W[8] = mk2(__uint_as_float(r.lt.x), __uint_as_float(r.lt.y));
    } else {
        W[0] = cvt_pair(r.l[0].x); W[1] = cvt_pair(r.l[0].y); W[2] = cvt_pair(r.l[0].z); W[3] = cvt_pair(r.l[0].w);
        if constexpr (RECON == 18) {
            W[4] = cvt_pair(r.l[1].x); W[5] = cvt_pair(r.l[1].y); W[6] = cvt_pair(r.l[1].z); W[7] = cvt_pair(r.l[1].w);
            W[8] = cvt_pair(r.lt.x);
        } else {
            W[4] = cvt_pair(r.lt.x); W[5] = cvt_pair(r.lt.y);
        }
    }
    if constexpr (RECON != 18) link_row2_f2(W);
}

// ---- a3: spin projection, packed ----------------------------------------------------------------------
// Every output pair is  U + c * L'  with c = +-1 per lane (L' = L, maybe lane-swapped).  BIASED (half): U and L carry
// the conversion bias M; a lane with c = -1 cancels it exactly, a lane with c = +1 needs U - 2M first (exact: all
// values are integers below 2^24), so the conversion costs one FADD2 per pair with a +1 lane instead of one per
// input pair, and the result is bit-identical to projecting the unbiased integers.
template <bool BIASED>
TM_DEV f2 proj_fma(f2 L, f2 c, f2 U)
{
    if constexpr (BIASED) {
        if (c.x > 0.f || c.y > 0.f) U = add2(U, mk2(c.x > 0.f ? -2.f * TM_CVT_MAGIC : 0.f, c.y > 0.f ? -2.f * TM_CVT_MAGIC : 0.f));
    }
    return fma2(L, c, U);
}
template <int MU, int SGN, bool BIASED = false>
TM_DEV void project_f2(f2 *H, const f2 *S)
{
    const f2 *U = S, *L = S + 6;
    const f2 pm = mk2((float)SGN, (float)-SGN), mp = mk2((float)-SGN, (float)SGN);
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const f2 Ur = U[2 * c], Ui = U[2 * c + 1], Lr = L[2 * c], Li = L[2 * c + 1];
        if constexpr (MU == 0) {
            H[2 * c] = proj_fma<BIASED>(sw2(Li), bc2((float)SGN), Ur);
            H[2 * c + 1] = proj_fma<BIASED>(sw2(Lr), bc2((float)-SGN), Ui);
        } else if constexpr (MU == 1) {
            H[2 * c] = proj_fma<BIASED>(sw2(Lr), mp, Ur);
            H[2 * c + 1] = proj_fma<BIASED>(sw2(Li), mp, Ui);
        } else {
            H[2 * c] = proj_fma<BIASED>(Li, pm, Ur);
            H[2 * c + 1] = proj_fma<BIASED>(Lr, mp, Ui);
        }
    }
}

// ---- a5: color multiply on both spin components at once: 36 packed instructions ------------------------
// Order: for every input colour d, the six accumulations that read H_re[d] one after the other, then the six that read H_im[d].
// Consecutive FFMA2 then share their pair operand, which ptxas serves from the register reuse cache: an FFMA2 with three distinct
// register sources occupies the sub-partition for 3 cycles, with a cached pair for 2 (profiles/r2_pipes.md).  The six accumulators of
// a group are independent, and every accumulator still sums its terms in the order d = 0, 1, 2 (re, im within d): same bits as before.
template <bool ADJ>
TM_DEV void su3_mul_f2(f2 *G, const f2 *W, const f2 *H)
{
    f2 re[3], im[3];
#pragma unroll
    for (int d = 0; d < 3; d++) {
        float ur[3], ui[3];
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const f2 w = ADJ ? W[3 * d + c] : W[3 * c + d];
            ur[c] = w.x;
            ui[c] = ADJ ? -w.y : w.y;
        }
        const f2 hr = H[2 * d], hi = H[2 * d + 1];
#pragma unroll
        for (int c = 0; c < 3; c++) re[c] = (d == 0) ? mul2(bc2(ur[c]), hr) : fma2(bc2(ur[c]), hr, re[c]);
#pragma unroll
        for (int c = 0; c < 3; c++) im[c] = (d == 0) ? mul2(bc2(ui[c]), hr) : fma2(bc2(ui[c]), hr, im[c]);
#pragma unroll
        for (int c = 0; c < 3; c++) re[c] = fma2(bc2(-ui[c]), hi, re[c]);
#pragma unroll
        for (int c = 0; c < 3; c++) im[c] = fma2(bc2(ur[c]), hi, im[c]);
    }
#pragma unroll
    for (int c = 0; c < 3; c++) {
        G[2 * c] = re[c];
        G[2 * c + 1] = im[c];
    }
}

// ---- a5: reconstruction + accumulate with weight w:  A_u += w G ;  A_l += w sgn i sigma_k G -----------
//   x: (i s1 g) = (i g1, i g0)  -> Alr += -sgn sw(Gi), Ali += +sgn sw(Gr)
//   y: (i s2 g) = (g1, -g0)     -> Alr += (sgn,-sgn) sw(Gr), Ali += (sgn,-sgn) sw(Gi)
//   z: (i s3 g) = (i g0, -i g1) -> Alr += (-sgn,sgn) Gi,     Ali += (sgn,-sgn) Gr
// w2 = the weight of color 2 (differs from w only when row 2 of a half-precision link was left unscaled).
template <int MU, int SGN>
TM_DEV void reconstruct_f2(f2 *A, const f2 *G, float w, float w2)
{
    f2 *Au = A, *Al = A + 6;
    if constexpr (MU == 3) {
        f2 *dst = (SGN > 0) ? Al : Au;
#pragma unroll
        for (int i = 0; i < 6; i++) dst[i] = fma2(G[i], bc2(i < 4 ? w : w2), dst[i]);
    } else {
#pragma unroll
        for (int i = 0; i < 6; i++) Au[i] = fma2(G[i], bc2(i < 4 ? w : w2), Au[i]);
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const float sw_ = (float)SGN * (c < 2 ? w : w2);
            const f2 pm = mk2(sw_, -sw_), mp = mk2(-sw_, sw_);
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

// Where the fields are: the same for every site of a launch (kept in uniform registers).
struct HopPtrs {
    const char *in;          // input spinor field
    const char *x;           // xpay input (own parity)
    const char *gf, *gb;     // gauge blocks of the output parity (forward links) / the other parity (backward links)
};
// a2: one output site: its checkerboard index, the 8 neighbour indices (periodic wrap) and the time-hop weights.
struct HopCtx {
    int site;
    int nbr[8];              // +x -x +y -y +z -z +t -t
    float wt[2];             // weight of the +t / -t hop (2 x boundary sign; 0 when the hop leaves a sub-lattice cut in t)
    float ws[4];             // weight of the +y -y +z -z hop (1; 0 when the hop leaves a sub-lattice cut in that direction)
};

TM_DEV void site_ctx(HopCtx &c, const DslashArgs &a, int site)
{
    const int Xh = a.Xh;
    int r = tm_div(site, a.dXh);
    const int xh = site - r * Xh;
    int r2 = tm_div(r, a.dY);
    const int y = r - r2 * a.Y;
    const int t = tm_div(r2, a.dZ);
    const int z = r2 - t * a.Z;
    const int q = (y + z + t + a.parity) & 1;       // x1 = 2 xh + q
    const int sy = Xh, sz = Xh * a.Y, st = Xh * a.Y * a.Z;
    c.site = site;
    c.nbr[0] = q ? ((xh + 1 == Xh) ? site - (Xh - 1) : site + 1) : site;
    c.nbr[1] = q ? site : ((xh == 0) ? site + (Xh - 1) : site - 1);
    c.nbr[2] = (y == a.Y - 1) ? site - (a.Y - 1) * sy : site + sy;
    c.nbr[3] = (y == 0) ? site + (a.Y - 1) * sy : site - sy;
    c.nbr[4] = (z == a.Z - 1) ? site - (a.Z - 1) * sz : site + sz;
    c.nbr[5] = (z == 0) ? site + (a.Z - 1) * sz : site - sz;
    c.nbr[6] = (t == a.T - 1) ? site - (a.T - 1) * st : site + st;
    c.nbr[7] = (t == 0) ? site + (a.T - 1) * st : site - st;
    c.wt[0] = 2.f * ((t == a.T - 1) ? (float)a.tbound : 1.f);
    c.wt[1] = 2.f * ((t == 0) ? (float)a.tbound : 1.f);
    c.ws[0] = (y == a.Y - 1) ? a.wrap_y : 1.f;
    c.ws[1] = (y == 0) ? a.wrap_y : 1.f;
    c.ws[2] = (z == a.Z - 1) ? a.wrap_z : 1.f;
    c.ws[3] = (z == 0) ? a.wrap_z : 1.f;
}

// Pipeline slot H of a site: 0..7 = the hops in the order of HopCtx::nbr, 8 = the xpay input of the site, > 8 nothing.
// One address computation per neighbour (spinor_site_off / link_site_off); every load then uses an immediate offset.
template <int PREC, int NF, int RECON, int KT, bool DAG, bool STG, int H, bool TWIN = false>
TM_DEV void issue_slot(HopRaw<PREC, NF, RECON> &r, const HopPtrs &p, const HopCtx &c)
{
    if constexpr (H < 8) {
        constexpr int MU = H / 2;
        constexpr bool FWD = (H % 2) == 0;
        constexpr int SGN = (FWD != DAG) ? +1 : -1;
        constexpr int PART = (MU == 3 && !TWIN) ? ((SGN > 0) ? 2 : 1) : 0;      // TWIN: the input twist needs the whole neighbour site
        const int n = c.nbr[H];
        if constexpr (!STG) {
            if constexpr (FWD) issue_link<PREC, NF, RECON, false>(r, p.gf + link_site_off(PREC, RECON, c.site, MU), c.site & (TM_TILE - 1));
            else issue_link<PREC, NF, RECON, false>(r, p.gb + link_site_off(PREC, RECON, n, MU), n & (TM_TILE - 1));
        }
        issue_spinor<PREC, NF, RECON, PART>(r, p.in + spinor_site_off(PREC, NF, n, 0), n & (TM_TILE - 1));
    } else if constexpr (H == 8 && KT != 0) {
        issue_spinor<PREC, NF, RECON, 0>(r, p.x + spinor_site_off(PREC, NF, c.site, 0), c.site & (TM_TILE - 1));
    }
}

template <int NF>
TM_DEV void twist_f2(f2 *Wo, const f2 *V, const f2 *O, float alpha, float beta, float scale);
struct TwistInF { float alpha, beta, scale; };      // the twist applied to the INPUT sites (TWIN kernels)

// a6: the link is converted and rebuilt once and applied to every flavor.
template <int PREC, int NF, int RECON, bool DAG, bool STG, int H, bool TWIN = false>
TM_DEV void consume_hop(f2 *A, HopRaw<PREC, NF, RECON> &r, const HopCtx &c, TwistInF ti = TwistInF())
{
    constexpr int MU = H / 2;
    constexpr bool FWD = (H % 2) == 0;
    constexpr int SGN = (FWD != DAG) ? +1 : -1;
    constexpr int PART = (MU == 3 && !TWIN) ? ((SGN > 0) ? 2 : 1) : 0;
    if constexpr (STG) {
        cp_async_wait<7 - H>();
        issue_link<PREC, NF, RECON, true>(r, stage_slot<PREC, RECON>(H), threadIdx.x & 31);
    }
    f2 W[9];
    raw_to_link<PREC, NF, RECON>(W, r);
    const float w = (MU == 3) ? c.wt[H & 1] : (MU == 0) ? 1.f : c.ws[H - 2];
    f2 T[TWIN ? NF * 12 : 1];
    if constexpr (TWIN) {
        // D R^-1: every flavor of the neighbour site at true scale (half: raw integers x norm / 32767), twisted in registers
        f2 V[NF * 12];
#pragma unroll
        for (int f = 0; f < NF; f++) {
            raw_to_spinor<PREC, 0>(V + 12 * f, r.s[f]);
            if constexpr (PREC == 2) {
                const float sc = r.n[f] * TM_INV15;
#pragma unroll
                for (int i = 0; i < 12; i++) V[12 * f + i] = mul2(V[12 * f + i], bc2(sc));
            }
        }
#pragma unroll
        for (int f = 0; f < NF; f++) twist_f2<NF>(T + 12 * f, V + 12 * f, V + 12 * (NF - 1 - f), f == 0 ? ti.alpha : -ti.alpha, ti.beta, ti.scale);
    }
#pragma unroll
    for (int f = 0; f < NF; f++) {
        f2 S[12], H6[6], G[6];
        if constexpr (TWIN) {
            if constexpr (MU == 3) {
#pragma unroll
                for (int i = 0; i < 6; i++) H6[i] = (SGN > 0) ? T[12 * f + 6 + i] : T[12 * f + i];
            } else {
                project_f2<MU, SGN>(H6, T + 12 * f);
            }
        } else if constexpr (MU == 3) {
            raw_to_spinor<PREC, PART>(S, r.s[f]);
#pragma unroll
            for (int i = 0; i < 6; i++) H6[i] = (SGN > 0) ? S[6 + i] : S[i];
        } else {
            raw_to_spinor<PREC, PART, PREC == 2>(S, r.s[f]);
            project_f2<MU, SGN, PREC == 2>(H6, S);
        }
        float wf = w, wf2 = w;
        if constexpr (PREC == 2) {
            // site norm x spinor scale (already applied when TWIN) x link scale (8-real links are rebuilt at true scale)
            wf *= (TWIN ? 1.f : r.n[f] * TM_INV15) * (RECON == 8 ? 1.f : TM_INV15);
            wf2 = wf;
            if constexpr (RECON == 12) {                                 // row 2 of the link carries an extra 32767
                if constexpr (FWD) wf2 = wf * TM_INV15;                  // U h: row 2 -> output color 2
                else { H6[4] = mul2(H6[4], bc2(TM_INV15)); H6[5] = mul2(H6[5], bc2(TM_INV15)); }   // U^+ h: row 2 meets h color 2
            }
        }
        su3_mul_f2<!FWD>(G, W, H6);
        reconstruct_f2<MU, SGN>(A + 12 * f, G, wf, wf2);
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
TM_DEV void store_spinor_f2(const f2 *A, char *sp, int lane)
{
    if constexpr (PREC == 4) {
#pragma unroll
        for (int k = 0; k < 6; k++)
            *reinterpret_cast<float4 *>(sp + k * TM_PLANE) = make_float4(A[2 * k].x, A[2 * k].y, A[2 * k + 1].x, A[2 * k + 1].y);
    } else {
        float m = 0.f;
#pragma unroll
        for (int i = 0; i < 12; i++) m = fmaxf(m, fmaxf(fabsf(A[i].x), fabsf(A[i].y)));
        const float s = (m > 0.f) ? __fdividef(32767.0f, m) : 0.f;
#pragma unroll
        for (int k = 0; k < 3; k++) {
            int4 c;
            c.x = quant_pair(A[4 * k], s);
            c.y = quant_pair(A[4 * k + 1], s);
            c.z = quant_pair(A[4 * k + 2], s);
            c.w = quant_pair(A[4 * k + 3], s);
            *reinterpret_cast<int4 *>(sp + k * TM_PLANE) = c;
        }
        *reinterpret_cast<float *>(sp + tail_off(3, 4, lane)) = m;
    }
}

// slot 8: the xpay input of the site, from raw words to values
template <int PREC, int NF, int RECON>
TM_DEV void load_x(f2 *X, const HopRaw<PREC, NF, RECON> &rx)
{
#pragma unroll
    for (int f = 0; f < NF; f++) {
        raw_to_spinor<PREC, 0>(X + 12 * f, rx.s[f]);
        if constexpr (PREC == 2) {
            const float s = rx.n[f] * TM_INV15;
#pragma unroll
            for (int i = 0; i < 12; i++) X[12 * f + i] = mul2(X[12 * f + i], bc2(s));
        }
    }
}

// One thread per output site, all flavors.  The 8 hops and the xpay input are 9 pipeline slots; slot h + PD is
// issued before hop h is computed (PD = f2_pipeline_depth, PD + 1 rotating raw buffers).
template <int PREC, int NF, int RECON, int KT, bool DAG, bool STG, bool TWIN = false>
__global__ void __launch_bounds__(128, f2_min_blocks<PREC, NF>()) tm_dslash_f2(const DslashArgs a)
{
    constexpr int PD = f2_pipeline_depth<PREC, NF>();
    tm_pdl_enter();
    const int Vh = a.Vh;
    const int vblock = tm_virtual_block(a, blockIdx.x);
    prefetch_tile<PREC, NF, RECON, KT != 0>(a, blockDim.x, vblock);
    const int site = vblock * blockDim.x + threadIdx.x;
    if (site >= Vh) return;

    HopPtrs p;
    const size_t PB = (size_t)tm_tiles(Vh) * 4 * link_tile_bytes(PREC, RECON);     // one parity's gauge block
    p.in = static_cast<const char *>(a.in);
    p.x = static_cast<const char *>(a.x);
    p.gf = static_cast<const char *>(a.gauge) + (size_t)a.parity * PB;
    p.gb = static_cast<const char *>(a.gauge) + (size_t)(1 - a.parity) * PB;

    HopCtx c;
    site_ctx(c, a, site);
    if constexpr (STG) {
#pragma unroll
        for (int h = 0; h < 8; h++)
            stage_link<PREC, RECON>(h, (h & 1) ? p.gb + link_site_off(PREC, RECON, c.nbr[h], h >> 1) : p.gf + link_site_off(PREC, RECON, site, h >> 1),
                                    ((h & 1) ? c.nbr[h] : site) & (TM_TILE - 1));
    }

    f2 A[NF * 12], X[NF * 12];
#pragma unroll
    for (int i = 0; i < NF * 12; i++) A[i] = mk2(0.f, 0.f);

    HopRaw<PREC, NF, RECON> buf[PD + 1];
    TwistInF ti;
    ti.alpha = (float)a.alpha_in; ti.beta = (float)a.beta_in; ti.scale = (float)a.scale_in;
#define TM_ISSUE(S) issue_slot<PREC, NF, RECON, KT, DAG, STG, (S), TWIN>(buf[(S) % (PD + 1)], p, c)
#define TM_STEP(H)                                                                  \
    do {                                                                            \
        TM_ISSUE((H) + PD);                                                         \
        consume_hop<PREC, NF, RECON, DAG, STG, (H), TWIN>(A, buf[(H) % (PD + 1)], c, ti);     \
    } while (0)
    if constexpr (PD >= 1) TM_ISSUE(0);
    if constexpr (PD >= 2) TM_ISSUE(1);
    if constexpr (PD >= 3) TM_ISSUE(2);
    TM_STEP(0); TM_STEP(1); TM_STEP(2); TM_STEP(3); TM_STEP(4); TM_STEP(5); TM_STEP(6); TM_STEP(7);
    if constexpr (PD == 0) TM_ISSUE(8);
#undef TM_STEP
#undef TM_ISSUE
    if constexpr (KT != 0) load_x<PREC, NF, RECON>(X, buf[8 % (PD + 1)]);

    epilogue_f2<NF, KT>(A, X, (float)a.alpha, (float)a.beta, (float)a.scale, (float)a.kappa, (float)a.kappa2);

    char *os = static_cast<char *>(a.out) + spinor_site_off(PREC, NF, site, 0);
#pragma unroll
    for (int f = 0; f < NF; f++) store_spinor_f2<PREC>(A + 12 * f, os + f * spinor_tile_bytes(PREC), site & (TM_TILE - 1));
}

template <int PREC, int NF, int RECON, int KT, bool DAG, bool STG, bool TWIN = false>
cudaError_t tm_launch_f2(const DslashArgs &a, cudaStream_t s)
{
    const int threads = a.block_threads;
    const int blocks = (a.Vh + threads - 1) / threads;
    const size_t smem = STG ? (size_t)8 * RECON * PREC * threads : 0;
    if (smem > 48 * 1024) {
        static std::atomic<unsigned long long> raised{0};      // per instantiation, one bit per device
        cudaError_t e = tm_raise_smem(tm_dslash_f2<PREC, NF, RECON, KT, DAG, STG, TWIN>, raised);
        if (e != cudaSuccess) return e;
    }
    return tm_launch_kernel(tm_dslash_f2<PREC, NF, RECON, KT, DAG, STG, TWIN>, a.pdl, blocks, threads, smem, s, a);
}

// table index: [recon18?0:1][kt 0..3][dagger 0..1][staged 0..1]
#define TM_F2_ROW(P, N, R, K)                                                                       \
    {tm_launch_f2<P, N, R, K, false, false>, "f2<" #P "," #N "," #R "," #K ",plain>"},             \
    {tm_launch_f2<P, N, R, K, false, true>, "f2_staged<" #P "," #N "," #R "," #K ",plain>"},       \
    {tm_launch_f2<P, N, R, K, true, false>, "f2<" #P "," #N "," #R "," #K ",dagger>"},             \
    {tm_launch_f2<P, N, R, K, true, true>, "f2_staged<" #P "," #N "," #R "," #K ",dagger>"}
// 8-real links: direct loads only (both staging slots hold the direct kernel)
#define TM_F2_ROW8(P, N, K)                                                                        \
    {tm_launch_f2<P, N, 8, K, false, false>, "f2<" #P "," #N ",8," #K ",plain>"},                 \
    {tm_launch_f2<P, N, 8, K, false, false>, "f2<" #P "," #N ",8," #K ",plain>"},                 \
    {tm_launch_f2<P, N, 8, K, true, false>, "f2<" #P "," #N ",8," #K ",dagger>"},                 \
    {tm_launch_f2<P, N, 8, K, true, false>, "f2<" #P "," #N ",8," #K ",dagger>"}
#define TM_F2_ROWS8(P, N) , TM_F2_ROW8(P, N, 0), TM_F2_ROW8(P, N, 1), TM_F2_ROW8(P, N, 2), TM_F2_ROW8(P, N, 3)
// input-twist (D R^-1) kernels, direct loads only: index [recon 18 / 12 / 8 -> 0 / 1 / 2][A, REC -> 0, 1][dagger 0..1]
#define TM_F2_TWIN_ROW(P, N, R)                                                                      \
    {tm_launch_f2<P, N, R, 0, false, false, true>, "f2_twin<" #P "," #N "," #R ",0,plain>"},        \
    {tm_launch_f2<P, N, R, 0, true, false, true>, "f2_twin<" #P "," #N "," #R ",0,dagger>"},        \
    {tm_launch_f2<P, N, R, 3, false, false, true>, "f2_twin<" #P "," #N "," #R ",3,plain>"},        \
    {tm_launch_f2<P, N, R, 3, true, false, true>, "f2_twin<" #P "," #N "," #R ",3,dagger>"}
#define TM_F2_TABLE(P, N)                                                                    \
    static const TmKernelEntry f2twin_##P##_##N[12] = {TM_F2_TWIN_ROW(P, N, 18), TM_F2_TWIN_ROW(P, N, 12), TM_F2_TWIN_ROW(P, N, 8)};   \
    const TmKernelEntry *tm_f2_twin_table_##P##_##N() { return f2twin_##P##_##N; }          \
    static const TmKernelEntry f2table_##P##_##N[48] = {                                    \
        TM_F2_ROW(P, N, 18, 0), TM_F2_ROW(P, N, 18, 1), TM_F2_ROW(P, N, 18, 2),             \
        TM_F2_ROW(P, N, 18, 3), TM_F2_ROW(P, N, 12, 0), TM_F2_ROW(P, N, 12, 1),             \
        TM_F2_ROW(P, N, 12, 2), TM_F2_ROW(P, N, 12, 3) TM_F2_ROWS8(P, N)};                 \
    const TmKernelEntry *tm_f2_table_##P##_##N() { return f2table_##P##_##N; }

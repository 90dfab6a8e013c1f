// tm_layout.cuh -- register <-> device-layout moves for spinors and links (rows a1, a4, a8 of DESIGN.md).
// A site's spinor is 24 reals v[(spin*3+color)*2+reim]; "upper" = spin 0,1 = v[0..11], "lower" = v[12..23].
// A link is 18 reals u[(row*3+col)*2+reim].
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#ifndef TM_DEV
#define TM_DEV __device__ __forceinline__
#endif

template <int PREC> struct PrecTraits;
template <> struct PrecTraits<8> { typedef double real; static constexpr int NCH = 12; };
template <> struct PrecTraits<4> { typedef float real;  static constexpr int NCH = 6; };
template <> struct PrecTraits<2> { typedef float real;  static constexpr int NCH = 3; };

#define TM_HALF_MAX 32767.0f
#define TM_HALF_INV (1.0f / 32767.0f)

// ---- tiled SoA addressing ----------------------------------------------------------
// Fields are cut into TILES of 32 consecutive checkerboard sites (one warp).  Inside a tile every 128-bit chunk is
// a PLANE of 32 x 16 = 512 contiguous bytes, so a warp's access to a plane is one 512-byte segment and the planes
// of a site are at COMPILE-TIME offsets from the site's pointer (one address computation per neighbour, immediate
// offsets for every further load).
//   spinor, one parity : [tile][flavor][plane][32]   planes: 12 (fp64) / 6 (fp32) / 3 + a 128-byte norm plane (half)
//   gauge              : [parity][tile][mu][plane][32]  planes of 16 bytes per site, then one narrower tail plane
#define TM_TILE 32
#define TM_TILE_LOG 5
#define TM_PLANE 512
__host__ __device__ constexpr int spinor_tile_bytes(int prec) { return prec == 8 ? 12 * 512 : prec == 4 ? 6 * 512 : 3 * 512 + 128; }
__host__ __device__ constexpr int link_tile_bytes(int prec, int recon) { return recon * prec * TM_TILE; }
__host__ __device__ inline int tm_tiles(int Vh) { return (Vh + TM_TILE - 1) / TM_TILE; }
// byte offset of (site idx, flavor f) in a spinor field of nf flavors: points at the site's 16 bytes of plane 0
__host__ __device__ inline size_t spinor_site_off(int prec, int nf, int idx, int f)
{
    return ((size_t)(idx >> TM_TILE_LOG) * nf + f) * spinor_tile_bytes(prec) + (size_t)(idx & (TM_TILE - 1)) * 16;
}
// byte offset of U_mu at site idx inside one parity's gauge block (block size = tiles * 4 * link_tile_bytes)
__host__ __device__ inline size_t link_site_off(int prec, int recon, int idx, int mu)
{
    return ((size_t)(idx >> TM_TILE_LOG) * 4 + mu) * link_tile_bytes(prec, recon) + (size_t)(idx & (TM_TILE - 1)) * 16;
}
// A narrower plane (w bytes per site) that follows n16 full planes: its element for `lane` relative to the site pointer
__host__ __device__ constexpr int tail_off(int n16, int w, int lane) { return n16 * TM_PLANE - lane * (16 - w); }

TM_DEV float tm_fma(float a, float b, float c) { return __fmaf_rn(a, b, c); }
TM_DEV double tm_fma(double a, double b, double c) { return __fma_rn(a, b, c); }

// ---- raw 128-bit global accesses ------------------------------------------------------------------
TM_DEV double2 ldg_d2(const void *p) { return __ldg(reinterpret_cast<const double2 *>(p)); }
TM_DEV float4 ldg_f4(const void *p) { return __ldg(reinterpret_cast<const float4 *>(p)); }
TM_DEV float2 ldg_f2(const void *p) { return __ldg(reinterpret_cast<const float2 *>(p)); }
TM_DEV int4 ldg_i4(const void *p) { return __ldg(reinterpret_cast<const int4 *>(p)); }
TM_DEV int2 ldg_i2(const void *p) { return __ldg(reinterpret_cast<const int2 *>(p)); }
TM_DEV int ldg_i1(const void *p) { return __ldg(reinterpret_cast<const int *>(p)); }
TM_DEV float ldg_f1(const void *p) { return __ldg(reinterpret_cast<const float *>(p)); }
// The gauge field is read exactly once per launch and is most of the traffic; the input spinor is read 8 times (once per
// neighbouring output site) over a window of two time slices.  On lattices whose time slice (both gauge parities + spinor) does
// not fit the 126 MB L2 next to the streaming links (48^3 x 96: ~85 MB of links per slice), the links evict the spinor before
// its reuse and DRAM traffic rises above the algorithmic bytes.  Link loads therefore carry an L2 evict-first policy
// (createpolicy + ld.global.nc.L2::cache_hint): they leave the L2 first, the spinor stays.
#ifndef TM_LINK_HINT
#define TM_LINK_HINT 1
#endif
TM_DEV unsigned long long tm_policy_stream()
{
    unsigned long long p;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
TM_DEV double2 ldg_stream_d2(const void *p)
{
#if TM_LINK_HINT
    double2 v;
    asm("ld.global.nc.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(tm_policy_stream()));
    return v;
#else
    return ldg_d2(p);
#endif
}
TM_DEV uint4 ldg_stream_u4(const void *p)
{
    uint4 v;
#if TM_LINK_HINT
    asm("ld.global.nc.L2::cache_hint.v4.u32 {%0, %1, %2, %3}, [%4], %5;" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p), "l"(tm_policy_stream()));
#else
    asm("ld.global.nc.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
#endif
    return v;
}
TM_DEV uint2 ldg_stream_u2(const void *p)
{
    uint2 v;
#if TM_LINK_HINT
    asm("ld.global.nc.L2::cache_hint.v2.u32 {%0, %1}, [%2], %3;" : "=r"(v.x), "=r"(v.y) : "l"(p), "l"(tm_policy_stream()));
#else
    asm("ld.global.nc.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
#endif
    return v;
}
TM_DEV unsigned ldg_stream_u1(const void *p)
{
    unsigned v;
#if TM_LINK_HINT
    asm("ld.global.nc.L2::cache_hint.u32 %0, [%1], %2;" : "=r"(v) : "l"(p), "l"(tm_policy_stream()));
#else
    asm("ld.global.nc.u32 %0, [%1];" : "=r"(v) : "l"(p));
#endif
    return v;
}
// link loads.  SM = true: the pointer is shared memory (staged links, tm_stream.cuh) -> plain loads; else streaming global loads
template <bool SM> TM_DEV double2 ld_d2(const void *p) { if constexpr (SM) return *reinterpret_cast<const double2 *>(p); else return ldg_stream_d2(p); }
template <bool SM> TM_DEV float4 ld_f4(const void *p)
{
    if constexpr (SM) return *reinterpret_cast<const float4 *>(p);
    else { const uint4 v = ldg_stream_u4(p); return make_float4(__uint_as_float(v.x), __uint_as_float(v.y), __uint_as_float(v.z), __uint_as_float(v.w)); }
}
template <bool SM> TM_DEV float2 ld_f2(const void *p)
{
    if constexpr (SM) return *reinterpret_cast<const float2 *>(p);
    else { const uint2 v = ldg_stream_u2(p); return make_float2(__uint_as_float(v.x), __uint_as_float(v.y)); }
}
template <bool SM> TM_DEV int4 ld_i4(const void *p)
{
    if constexpr (SM) return *reinterpret_cast<const int4 *>(p);
    else { const uint4 v = ldg_stream_u4(p); return make_int4((int)v.x, (int)v.y, (int)v.z, (int)v.w); }
}
template <bool SM> TM_DEV int2 ld_i2(const void *p)
{
    if constexpr (SM) return *reinterpret_cast<const int2 *>(p);
    else { const uint2 v = ldg_stream_u2(p); return make_int2((int)v.x, (int)v.y); }
}
template <bool SM> TM_DEV int ld_i1(const void *p) { if constexpr (SM) return *reinterpret_cast<const int *>(p); else return (int)ldg_stream_u1(p); }

// Stored int16 are OFFSET BINARY (u = q + 32768, see tm_f2.cuh): two per 32-bit word -> two floats (exact), times s
TM_DEV void unpack2(int w, float s, float &lo, float &hi)
{
    lo = (float)((int)(w & 0xffff) - 32768) * s;
    hi = (float)((int)((unsigned)w >> 16) - 32768) * s;
}
TM_DEV int pack2(float lo, float hi)
{
    int a = __float2int_rn(lo) + 32768, b = __float2int_rn(hi) + 32768;
    return (a & 0xffff) | (b << 16);
}

// fp32 / half spinors keep a site's 24 reals in the order [half u/l][color][re/im][spin within the half], so that a
// 64-bit register pair holds the same (color, re/im) of two spin components (the packed-FP32 kernels, tm_f2.cuh).
// raw_pos(o): position in that order of the canonical real o = (spin*3+color)*2+reim.  fp64 stays canonical.
__host__ __device__ constexpr int raw_pos(int o)
{
    return ((o / 6) / 2) * 12 + ((o / 2) % 3) * 4 + (o % 2) * 2 + ((o / 6) % 2);
}

// ---- spinor loads ---------------------------------------------------------------------------------
// `sp` = the site's pointer (field + spinor_site_off), `lane` = idx & 31 (needed for the half norm plane).
// PART: 0 = all 24 reals, 1 = upper only (v[0..11] valid), 2 = lower only (v[12..23] valid).
template <int PART>
TM_DEV void load_spinor_half_raw(float *v, const char *sp, int lane);

template <int PREC, int PART>
TM_DEV void load_spinor(typename PrecTraits<PREC>::real *v, const char *sp, int lane)
{
    if constexpr (PREC == 8) {
        constexpr int lo = (PART == 2) ? 6 : 0, hi = (PART == 1) ? 6 : 12;
#pragma unroll
        for (int k = lo; k < hi; k++) {
            double2 c = ldg_d2(sp + k * TM_PLANE);
            v[2 * k] = c.x;
            v[2 * k + 1] = c.y;
        }
    } else if constexpr (PREC == 4) {
        constexpr int lo = (PART == 2) ? 3 : 0, hi = (PART == 1) ? 3 : 6;
        float r[24];
#pragma unroll
        for (int k = lo; k < hi; k++) {
            float4 c = ldg_f4(sp + k * TM_PLANE);
            r[4 * k] = c.x;
            r[4 * k + 1] = c.y;
            r[4 * k + 2] = c.z;
            r[4 * k + 3] = c.w;
        }
#pragma unroll
        for (int o = (PART == 2 ? 12 : 0); o < (PART == 1 ? 12 : 24); o++) v[o] = r[raw_pos(o)];
    } else {
        // 3 chunks of 8 int16: raw 0..7, 8..15, 16..23.  upper = raw 0..11, lower = raw 12..23.
        float r[24];
        load_spinor_half_raw<PART>(r, sp, lane);
#pragma unroll
        for (int o = (PART == 2 ? 12 : 0); o < (PART == 1 ? 12 : 24); o++) v[o] = r[raw_pos(o)];
    }
}

template <int PART>
TM_DEV void load_spinor_half_raw(float *v, const char *sp, int lane)
{
    const float s = ldg_f1(sp + tail_off(3, 4, lane)) * TM_HALF_INV;
    if constexpr (PART != 2) {
        int4 c = ldg_i4(sp);
        unpack2(c.x, s, v[0], v[1]);
        unpack2(c.y, s, v[2], v[3]);
        unpack2(c.z, s, v[4], v[5]);
        unpack2(c.w, s, v[6], v[7]);
    }
    {
        int4 c = ldg_i4(sp + TM_PLANE);
        if constexpr (PART != 2) {
            unpack2(c.x, s, v[8], v[9]);
            unpack2(c.y, s, v[10], v[11]);
        }
        if constexpr (PART != 1) {
            unpack2(c.z, s, v[12], v[13]);
            unpack2(c.w, s, v[14], v[15]);
        }
    }
    if constexpr (PART != 1) {
        int4 c = ldg_i4(sp + 2 * TM_PLANE);
        unpack2(c.x, s, v[16], v[17]);
        unpack2(c.y, s, v[18], v[19]);
        unpack2(c.z, s, v[20], v[21]);
        unpack2(c.w, s, v[22], v[23]);
    }
}

// ---- spinor store (a8): one write of the output site; half: norm = max|v|, q = rint(v * 32767 / norm)
template <int PREC>
TM_DEV void store_spinor(const typename PrecTraits<PREC>::real *v, char *sp, int lane)
{
    if constexpr (PREC == 8) {
#pragma unroll
        for (int k = 0; k < 12; k++) *reinterpret_cast<double2 *>(sp + k * TM_PLANE) = make_double2(v[2 * k], v[2 * k + 1]);
    } else if constexpr (PREC == 4) {
        float r[24];
#pragma unroll
        for (int o = 0; o < 24; o++) r[raw_pos(o)] = v[o];
#pragma unroll
        for (int k = 0; k < 6; k++)
            *reinterpret_cast<float4 *>(sp + k * TM_PLANE) = make_float4(r[4 * k], r[4 * k + 1], r[4 * k + 2], r[4 * k + 3]);
    } else {
        float r[24];
#pragma unroll
        for (int o = 0; o < 24; o++) r[raw_pos(o)] = v[o];
        v = r;
        float m = 0.f;
#pragma unroll
        for (int i = 0; i < 24; i++) m = fmaxf(m, fabsf(v[i]));
        const float s = (m > 0.f) ? __fdividef(TM_HALF_MAX, m) : 0.f;
#pragma unroll
        for (int k = 0; k < 3; k++) {
            int4 c;
            c.x = pack2(v[8 * k + 0] * s, v[8 * k + 1] * s);
            c.y = pack2(v[8 * k + 2] * s, v[8 * k + 3] * s);
            c.z = pack2(v[8 * k + 4] * s, v[8 * k + 5] * s);
            c.w = pack2(v[8 * k + 6] * s, v[8 * k + 7] * s);
            *reinterpret_cast<int4 *>(sp + k * TM_PLANE) = c;
        }
        *reinterpret_cast<float *>(sp + tail_off(3, 4, lane)) = m;
    }
}

// ---- link load + SU(3) row rebuild (a4) -----------------------------------------------------------
// 12-real: rows 0,1 stored, row2 = conj(row0 x row1).
template <typename real>
TM_DEV void rebuild_row2(real *u)
{
    // u[r][c] = u[(r*3+c)*2 + ri];  row2[c] = conj(row0[c+1] row1[c+2] - row0[c+2] row1[c+1])
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
        const real ar = u[2 * c1], ai = u[2 * c1 + 1];               // row0[c1]
        const real br = u[2 * (3 + c2)], bi = u[2 * (3 + c2) + 1];   // row1[c2]
        const real cr = u[2 * c2], ci = u[2 * c2 + 1];               // row0[c2]
        const real dr = u[2 * (3 + c1)], di = u[2 * (3 + c1) + 1];   // row1[c1]
        // explicit FMA chains: 4 + 4 instructions per component
        u[2 * (6 + c)] = tm_fma(ci, di, tm_fma(-cr, dr, tm_fma(-ai, bi, ar * br)));
        u[2 * (6 + c) + 1] = tm_fma(ci, dr, tm_fma(cr, di, tm_fma(-ai, br, -(ar * bi))));
    }
}

// 8-real ("8 or 12 parameter reconstruct"; the chart is DESIGN.md reading C11).  Stored, with rows a, b, c:
//   p[0..5] = a2, a3, b1 (re, im)   p[6] = arg(a1) / pi   p[7] = arg(c1) / pi      (all in [-1, 1])
// Rebuilt:  N = |a2|^2 + |a3|^2,  a1 = sqrt(1 - N) e^{i pi p6},  c1 = sqrt(N - |b1|^2) e^{i pi p7}  (row 0 and column 0
// have unit norm), then the two linear conditions  <a, b> = 0  and  c1 = conj(a2 b3 - a3 b2)  give
//   b2 = (r1 a2 - conj(a3) r2) / N ,  b3 = (conj(a2) r2 + a3 r1) / N ,   r1 = -conj(a1) b1 ,  r2 = conj(c1),
// and row 2 = conj(row0 x row1) as for 12-real.  The chart is singular at N = 0 (tm_gauge_load refuses such links).
TM_DEV void tm_sincospi(float x, float *s, float *c) { sincospif(x, s, c); }
TM_DEV float tm_sqrt_pos(float x) { return sqrtf(x); }
TM_DEV float tm_rcp(float x) { return 1.f / x; }
// fp64: branch-free forms (the library sincospi / sqrt / division carry slow paths and made the 8-real kernel FP64-pipe
// and branch bound).  |x| <= 1: q = rint(2x), r = x - q/2 in [-1/4, 1/4] (exact), Taylor polynomials of sin(pi r) and
// cos(pi r) to r^17 / r^18 (truncation < 1e-19), then the quadrant rotation.  Max error ~2e-16.
TM_DEV void tm_sincospi(double x, double *s, double *c)
{
    const double q = rint(x + x);
    const double r = fma(q, -0.5, x), r2 = r * r;
    const double S[9] = {3.14159265358979312e+00, -5.16771278004996937e+00, 2.55016403987734508e+00, -5.99264529320791883e-01, 8.21458866111281910e-02, -7.37043094571434784e-03, 4.66302805767612337e-04, -2.19153534478302037e-05, 7.95205400147550838e-07};
    const double C[10] = {1.00000000000000000e+00, -4.93480220054467900e+00, 4.05871212641676760e+00, -1.33526276885458928e+00, 2.35330630358893123e-01, -2.58068913900140508e-02, 1.92957430940392206e-03, -1.04638104924845650e-04, 4.30306958703294391e-06, -1.38789524622137608e-07};
    double ps = S[8], pc = C[9];
#pragma unroll
    for (int k = 7; k >= 0; k--) ps = fma(ps, r2, S[k]);
#pragma unroll
    for (int k = 8; k >= 0; k--) pc = fma(pc, r2, C[k]);
    ps *= r;
    const int iq = (int)q;                       // -2 .. 2
    const double a = (iq & 1) ? pc : ps, b = (iq & 1) ? ps : pc;      // sin, cos before the signs
    *s = (iq & 2) ? -a : a;
    *c = ((iq + 1) & 2) ? -b : b;
}
// sqrt(x) for x >= 0 and 1/x for x > 0 from the approximate units + two Newton steps (relative error ~1e-16)
TM_DEV double tm_sqrt_pos(double x)
{
    const double xs = fmax(x, 1e-300);
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(xs));
    y = y * fma(-0.5 * xs * y, y, 1.5);
    y = y * fma(-0.5 * xs * y, y, 1.5);
    const double r = x * y;                       // ~ sqrt(x); one correction step on the root itself
    return fma(0.5 * y, fma(-r, r, x), r);
}
TM_DEV double tm_rcp(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    y = y * fma(-x, y, 2.0);
    y = y * fma(-x, y, 2.0);
    return y * fma(-x, y, 2.0);
}
template <typename real>
TM_DEV void rebuild_from8(real *u, const real *p)
{
    const real a2r = p[0], a2i = p[1], a3r = p[2], a3i = p[3], b1r = p[4], b1i = p[5];
    const real N = tm_fma(a2r, a2r, tm_fma(a2i, a2i, tm_fma(a3r, a3r, a3i * a3i)));
    real s1, c1, s2, c2;
    tm_sincospi(p[6], &s1, &c1);
    tm_sincospi(p[7], &s2, &c2);
    const real m1 = tm_sqrt_pos(max((real)1 - N, (real)0));
    const real m2 = tm_sqrt_pos(max(N - tm_fma(b1r, b1r, b1i * b1i), (real)0));
    const real a1r = m1 * c1, a1i = m1 * s1;
    const real r2r = m2 * c2, r2i = -(m2 * s2);                               // conj(c1)
    const real r1r = -tm_fma(a1r, b1r, a1i * b1i), r1i = tm_fma(a1i, b1r, -(a1r * b1i));   // -conj(a1) b1
    const real iN = tm_rcp(N);
    u[0] = a1r; u[1] = a1i; u[2] = a2r; u[3] = a2i; u[4] = a3r; u[5] = a3i;
    u[6] = b1r; u[7] = b1i;
    u[8] = (tm_fma(r1r, a2r, -(r1i * a2i)) - tm_fma(a3r, r2r, a3i * r2i)) * iN;
    u[9] = (tm_fma(r1r, a2i, r1i * a2r) - tm_fma(a3r, r2i, -(a3i * r2r))) * iN;
    u[10] = (tm_fma(a2r, r2r, a2i * r2i) + tm_fma(a3r, r1r, -(a3i * r1i))) * iN;
    u[11] = (tm_fma(a2r, r2i, -(a2i * r2r)) + tm_fma(a3r, r1i, a3i * r1r)) * iN;
    rebuild_row2(u);
}

// Planes of a stored link: n16 planes of 16 bytes per site, then (maybe) one tail plane of `tailw` bytes per site.
template <int PREC, int RECON> __host__ __device__ constexpr int link_n16()
{
    return PREC == 8 ? RECON / 2 : PREC == 4 ? (RECON == 18 ? 4 : RECON == 12 ? 3 : 2) : (RECON == 18 ? 2 : 1);
}
template <int PREC, int RECON> __host__ __device__ constexpr int link_tailw()
{
    return PREC == 8 ? 0 : PREC == 4 ? (RECON == 18 ? 8 : 0) : (RECON == 18 ? 4 : RECON == 12 ? 8 : 0);
}

// `lp` = the link's site pointer (gauge parity block + link_site_off) or, SM = true, the thread's slot in the staged
// shared-memory copy, which keeps the same [plane][32 sites] shape per warp.
template <int PREC, int RECON, bool SM = false>
TM_DEV void load_link(typename PrecTraits<PREC>::real *u, const char *lp, int lane)
{
    constexpr int N16 = link_n16<PREC, RECON>();
    if constexpr (RECON == 8) {
        typename PrecTraits<PREC>::real p[8];
        if constexpr (PREC == 8) {
#pragma unroll
            for (int k = 0; k < 4; k++) {
                double2 c = ld_d2<SM>(lp + k * TM_PLANE);
                p[2 * k] = c.x;
                p[2 * k + 1] = c.y;
            }
        } else if constexpr (PREC == 4) {
#pragma unroll
            for (int k = 0; k < 2; k++) {
                float4 c = ld_f4<SM>(lp + k * TM_PLANE);
                p[4 * k] = c.x;
                p[4 * k + 1] = c.y;
                p[4 * k + 2] = c.z;
                p[4 * k + 3] = c.w;
            }
        } else {
            int4 c = ld_i4<SM>(lp);
            unpack2(c.x, TM_HALF_INV, p[0], p[1]);
            unpack2(c.y, TM_HALF_INV, p[2], p[3]);
            unpack2(c.z, TM_HALF_INV, p[4], p[5]);
            unpack2(c.w, TM_HALF_INV, p[6], p[7]);
        }
        rebuild_from8(u, p);
    } else if constexpr (PREC == 8) {
#pragma unroll
        for (int k = 0; k < N16; k++) {
            double2 c = ld_d2<SM>(lp + k * TM_PLANE);
            u[2 * k] = c.x;
            u[2 * k + 1] = c.y;
        }
    } else if constexpr (PREC == 4) {
#pragma unroll
        for (int k = 0; k < N16; k++) {
            float4 c = ld_f4<SM>(lp + k * TM_PLANE);
            u[4 * k] = c.x;
            u[4 * k + 1] = c.y;
            u[4 * k + 2] = c.z;
            u[4 * k + 3] = c.w;
        }
        if constexpr (RECON == 18) {
            float2 c = ld_f2<SM>(lp + tail_off(4, 8, lane));
            u[16] = c.x;
            u[17] = c.y;
        }
    } else {
        const float s = TM_HALF_INV;
        int4 c = ld_i4<SM>(lp);
        unpack2(c.x, s, u[0], u[1]);
        unpack2(c.y, s, u[2], u[3]);
        unpack2(c.z, s, u[4], u[5]);
        unpack2(c.w, s, u[6], u[7]);
        if constexpr (RECON == 18) {
            int4 d = ld_i4<SM>(lp + TM_PLANE);
            unpack2(d.x, s, u[8], u[9]);
            unpack2(d.y, s, u[10], u[11]);
            unpack2(d.z, s, u[12], u[13]);
            unpack2(d.w, s, u[14], u[15]);
            int e = ld_i1<SM>(lp + tail_off(2, 4, lane));
            unpack2(e, s, u[16], u[17]);
        } else {
            int2 d = ld_i2<SM>(lp + tail_off(1, 8, lane));
            unpack2(d.x, s, u[8], u[9]);
            unpack2(d.y, s, u[10], u[11]);
        }
    }
    if constexpr (RECON == 12) rebuild_row2(u);
}

TM_DEV void prefetch_l2(const void *p, unsigned bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// tm_dslash_tile.cuh -- the fused twisted-mass dslash for half precision with ONE WARP PER TILE and every operand of the warp
// staged through shared memory by asynchronous copies (rows a2-a9 of DESIGN.md).
//
// Why (profiles/r2_pipes.md): the half kernels are bound by the FP32 / integer datapath, and ~320 of their ~1550 instructions per
// site are address arithmetic -- a 64-bit address per neighbour spinor, norm, link and link tail, per thread.  In the tiled layout
// (tm_layout.cuh) the 32 sites of a warp are one tile, and the neighbours of a whole tile in the y, z, t directions are again whole
// tiles (z, t) or two half tiles (y), at warp-UNIFORM offsets; the x neighbours live in the tile of the same index.  So the warp
//   1. issues cp.async copies of the 6 (7) spinor tiles and the 8 link tiles it needs: per copy a warp-uniform tile base + lane * 16,
//      nothing site-specific, in four commit groups (x, y, z, t) so that the hops start while the later groups are still in flight;
//   2. computes the 8 hops from shared memory: the neighbour of lane l is slot l of the staged tile (z, t), slot l +- X/2 of the own
//      tile or of the assembled y-tile (y), slot l, l +- 1 with the row wrap (x): LDS with 32-bit addresses and immediate offsets.
// The arithmetic (conversion, projection, colour multiply, reconstruction, epilogue, quantisation) is tm_dslash_f2.cuh's, unchanged.
// Geometry: X/2 in {4, 8, 16} (a tile is R = 32 / (X/2) full x-rows), Y a multiple of R, V/2 a multiple of 32; other lattices
// take the thread-per-site kernels.  One block = one warp: every tile index is a function of blockIdx (uniform datapath).
#pragma once
#include "tm_dslash_f2.cuh"

struct TileGeom {
    int Xh, R, lg;         // sites per x-row of one parity (= 1 << lg); x-rows per tile
    int tps;               // tiles per (z, t) slab = Y / R
    TmFastDiv dtps, dZ;    // tile -> (slab, tile within slab); slab -> (t, z)
    const void *gauge_f, *gauge_b;   // the gauge blocks of the output parity / of the other parity
};

#ifndef TM_TILE_MINB_1
#define TM_TILE_MINB_1 12
#endif
#ifndef TM_TILE_MINB_2
#define TM_TILE_MINB_2 9
#endif

// ---- asynchronous copies of a tile: every lane moves 16 bytes per plane ---------------------------------------------------------
// `src` = the tile's address in global memory PLUS lane * 16, `dst` = the tile's shared-memory address plus lane * 16: one 64-bit
// address per (tile, lane) serves every plane through immediate offsets.  The narrow planes (norms: 4 bytes per site; link tails: 8
// or 4) are moved in 16-byte pieces too, by the first 8 or 16 lanes, so that they need no address of their own.
// PART: 0 all planes, 1 upper spin half only, 2 lower half only (half precision: planes {0,1} / {1,2}; the norm always)
template <int PREC, int PART>
TM_DEV void tile_copy_spinor_planes(unsigned dst, const char *src)
{
    static_assert(PREC == 2, "the tile kernel is instantiated for half precision");
    if constexpr (PART != 2) cp_async_u32<16>(dst, src);
    cp_async_u32<16>(dst + TM_PLANE, src + TM_PLANE);
    if constexpr (PART != 1) cp_async_u32<16>(dst + 2 * TM_PLANE, src + 2 * TM_PLANE);
}
TM_DEV void tile_copy_spinor_norms(unsigned dst, const char *src, int lane)      // 32 floats = 8 pieces
{
    if (lane < 8) cp_async_u32<16>(dst + 3 * TM_PLANE, src + 3 * TM_PLANE);
}
template <int PREC, int PART>
TM_DEV void tile_copy_spinor(unsigned dst, const char *src, int lane)
{
    tile_copy_spinor_planes<PREC, PART>(dst, src);
    tile_copy_spinor_norms(dst, src, lane);
}
// the time hops need one spin half (PART 1: planes 0, 1; PART 2: planes 1, 2): two planes and the norms, packed into TM_HALF_TILE bytes
constexpr int TM_HALF_TILE = 2 * TM_PLANE + TM_TILE * 4;
template <int PREC, int PART>
TM_DEV void tile_copy_half_spinor(unsigned dst, const char *src, int lane)
{
    static_assert(PREC == 2 && (PART == 1 || PART == 2), "half precision, one spin half");
    constexpr int K0 = PART == 1 ? 0 : 1;
    cp_async_u32<16>(dst, src + K0 * TM_PLANE);
    cp_async_u32<16>(dst + TM_PLANE, src + (K0 + 1) * TM_PLANE);
    if (lane < 8) cp_async_u32<16>(dst + 2 * TM_PLANE, src + 3 * TM_PLANE);
}
template <int PREC, int RECON>
TM_DEV void tile_copy_link_planes(unsigned dst, const char *src)
{
    constexpr int N16 = link_n16<PREC, RECON>();
#pragma unroll
    for (int k = 0; k < N16; k++) cp_async_u32<16>(dst + k * TM_PLANE, src + k * TM_PLANE);
}
template <int PREC, int RECON>
TM_DEV void tile_copy_link_tail(unsigned dst, const char *src, int lane)          // 32 x 8 bytes = 16 pieces, 32 x 4 bytes = 8 pieces
{
    constexpr int N16 = link_n16<PREC, RECON>(), TW = link_tailw<PREC, RECON>();
    if constexpr (TW > 0) {
        if (lane < 2 * TW) cp_async_u32<16>(dst + N16 * TM_PLANE, src + N16 * TM_PLANE);
    }
}
template <int PREC, int RECON>
TM_DEV void tile_copy_link(unsigned dst, const char *src, int lane)
{
    tile_copy_link_planes<PREC, RECON>(dst, src);
    tile_copy_link_tail<PREC, RECON>(dst, src, lane);
}

// ---- shared memory -> the raw words of one hop (what issue_link / issue_spinor load from global memory) ---------------------
TM_DEV uint4 lds_u4(unsigned a) { uint4 v; asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a)); return v; }
TM_DEV uint2 lds_u2(unsigned a) { uint2 v; asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a)); return v; }
TM_DEV unsigned lds_u1(unsigned a) { unsigned v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a)); return v; }

template <int PREC, int NF, int RECON>
TM_DEV void tile_read_spinor(HopRaw<PREC, NF, RECON> &r, unsigned stile, int slot)
{
    constexpr int STB = spinor_tile_bytes(PREC);
#pragma unroll
    for (int f = 0; f < NF; f++) {
        const unsigned p = stile + f * STB;
#pragma unroll
        for (int k = 0; k < 3; k++) r.s[f][k] = lds_u4(p + k * TM_PLANE + slot * 16);
        r.n[f] = __uint_as_float(lds_u1(p + 3 * TM_PLANE + slot * 4));
    }
}

template <int PREC, int NF, int RECON, int PART>
TM_DEV void tile_read_hop(HopRaw<PREC, NF, RECON> &r, unsigned stile, unsigned ltile, int sslot, int lslot)
{
    constexpr int STB = spinor_tile_bytes(PREC);
    r.l[0] = lds_u4(ltile + lslot * 16);
    if constexpr (RECON == 18) { r.l[1] = lds_u4(ltile + TM_PLANE + lslot * 16); r.lt.x = lds_u1(ltile + 2 * TM_PLANE + lslot * 4); }
    else r.lt = lds_u2(ltile + TM_PLANE + lslot * 8);
#pragma unroll
    for (int f = 0; f < NF; f++) {
        if constexpr (PART == 0) {
            const unsigned p = stile + f * STB;
#pragma unroll
            for (int k = 0; k < 3; k++) r.s[f][k] = lds_u4(p + k * TM_PLANE + sslot * 16);
            r.n[f] = __uint_as_float(lds_u1(p + 3 * TM_PLANE + sslot * 4));
        } else {                                                   // a packed half tile (tile_copy_half_spinor)
            constexpr int K0 = PART == 1 ? 0 : 1;
            const unsigned p = stile + f * TM_HALF_TILE;
            r.s[f][K0] = lds_u4(p + sslot * 16);
            r.s[f][K0 + 1] = lds_u4(p + TM_PLANE + sslot * 16);
            r.n[f] = __uint_as_float(lds_u1(p + 2 * TM_PLANE + sslot * 4));
        }
    }
}

template <int PREC, int NF, int RECON, int KT, bool DAG>
__global__ void __launch_bounds__(32, NF == 1 ? TM_TILE_MINB_1 : TM_TILE_MINB_2) tm_dslash_tile(const DslashArgs a, const TileGeom tg)
{
    constexpr int STB = spinor_tile_bytes(PREC), LTB = link_tile_bytes(PREC, RECON);
    constexpr int FS = NF * STB;                                   // all flavors of one spinor tile
    // shared memory of the warp: four spinor tiles (own index, assembled y, +z, -z), two half tiles (+t, -t), the 4 forward link tiles, 4 backward ones
    const unsigned sm = smem_u32(tm_smem);
    const unsigned SX = sm, SY = sm + FS, SZP = sm + 2 * FS, SZM = sm + 3 * FS, STP = sm + 4 * FS, STM = STP + NF * TM_HALF_TILE;
    const unsigned LF = STM + NF * TM_HALF_TILE, LBX = LF + 4 * LTB, LBY = LBX + LTB, LBZ = LBY + LTB, LBT = LBZ + LTB;

    // a2, per warp: the tile's place on the lattice and its neighbour tiles (functions of blockIdx: uniform)
    const int T = blockIdx.x, l = threadIdx.x;
    tm_pdl_enter();
    const int Xh = tg.Xh, R = tg.R, tps = tg.tps;
    const int slab = tps == 1 ? T : tm_div(T, tg.dtps), tin = T - slab * tps;
    const int t = tm_div(slab, tg.dZ), z = slab - t * a.Z;
    const int sz = tps, st = tps * a.Z;
    const int Tzp = (z == a.Z - 1) ? T - (a.Z - 1) * sz : T + sz, Tzm = (z == 0) ? T + (a.Z - 1) * sz : T - sz;
    const int Ttp = (t == a.T - 1) ? T - (a.T - 1) * st : T + st, Ttm = (t == 0) ? T + (a.T - 1) * st : T - st;
    const int Typ = (tin == tps - 1) ? T - (tps - 1) : T + 1, Tym = (tin == 0) ? T + (tps - 1) : T - 1;
    // per lane: row within the tile, x index, checkerboard offset
    const int row = l >> tg.lg, xh = l & (Xh - 1);
    const int y = tin * R + row;
    const int q = (y + z + t + a.parity) & 1;

    // per-lane 64-bit bases with the lane's 16 bytes folded in: a tile's address is then ONE multiply-add (tile index x tile bytes + base)
    const char *in_l = static_cast<const char *>(a.in) + l * 16;
    const char *gf_l = static_cast<const char *>(tg.gauge_f) + l * 16;     // forward links: the block of the output parity
    const char *gb_l = static_cast<const char *>(tg.gauge_b) + l * 16;     // backward links: the other parity's block
    // (opaque to the compiler, which otherwise keeps the pointer uniform and pays a 64-bit add per tile for the lane offset)
    asm volatile("" : "+l"(in_l), "+l"(gf_l), "+l"(gb_l));
    const unsigned sl = l * 16;
    auto spinor_tile = [&](int tile) { return in_l + (size_t)(unsigned)tile * FS; };
    auto link_tile = [&](const char *g, int tile, int mu) { return g + (size_t)(unsigned)(tile * 4 + mu) * LTB; };

    // ---- 1. every operand of the warp on its way to shared memory: four commit groups, in the order the hops consume them
    {
        const char *s0 = spinor_tile(T);
#pragma unroll
        for (int f = 0; f < NF; f++) tile_copy_spinor<PREC, 0>(SX + f * STB + sl, s0 + f * STB, l);
        const char *l0 = link_tile(gf_l, T, 0);
#pragma unroll
        for (int mu = 0; mu < 4; mu++) tile_copy_link<PREC, RECON>(LF + mu * LTB + sl, l0 + mu * LTB, l);
        tile_copy_link<PREC, RECON>(LBX + sl, link_tile(gb_l, T, 0), l);
    }
    cp_async_commit();
    {   // the y-tile: slots [0, Xh) from the tile after this one, slots [32 - Xh, 32) from the tile before (Xh = 16: every lane copies)
        const bool lo = l < Xh, hi = l >= 32 - Xh;
        if (lo || hi) {
            const char *sy = spinor_tile(lo ? Typ : Tym);
#pragma unroll
            for (int f = 0; f < NF; f++) tile_copy_spinor_planes<PREC, 0>(SY + f * STB + sl, sy + f * STB);
        }
        {   // its norms in 16-byte pieces of 4 slots (Xh is a multiple of 4: a piece never straddles the two source tiles)
            const bool nlo = 4 * l < Xh, nhi = 4 * l >= 32 - Xh;
            if (l < 8 && (nlo || nhi)) {
                const char *sn = spinor_tile(nlo ? Typ : Tym);
#pragma unroll
                for (int f = 0; f < NF; f++) cp_async_u32<16>(SY + f * STB + 3 * TM_PLANE + sl, sn + f * STB + 3 * TM_PLANE);
            }
        }
        // backward y links: U_y(x - y) sits at the neighbour's index: slots [0, 32 - Xh) in this tile, the rest in the tile before
        tile_copy_link_planes<PREC, RECON>(LBY + sl, link_tile(gb_l, (l < 32 - Xh) ? T : Tym, 1));
        constexpr int SPP = 16 / (link_tailw<PREC, RECON>() > 0 ? link_tailw<PREC, RECON>() : 16);      // slots per 16-byte tail piece
        tile_copy_link_tail<PREC, RECON>(LBY + sl, link_tile(gb_l, (SPP * l < 32 - Xh) ? T : Tym, 1), l);
    }
    cp_async_commit();
    {
        const char *zp = spinor_tile(Tzp), *zm = spinor_tile(Tzm);
#pragma unroll
        for (int f = 0; f < NF; f++) {
            tile_copy_spinor<PREC, 0>(SZP + f * STB + sl, zp + f * STB, l);
            tile_copy_spinor<PREC, 0>(SZM + f * STB + sl, zm + f * STB, l);
        }
        tile_copy_link<PREC, RECON>(LBZ + sl, link_tile(gb_l, Tzm, 2), l);
    }
    cp_async_commit();
    {   // a3: the time hops need half a spinor: (1 - gamma_4) keeps the lower half, (1 + gamma_4) the upper
        const char *tp = spinor_tile(Ttp), *tmn = spinor_tile(Ttm);
#pragma unroll
        for (int f = 0; f < NF; f++) {
            tile_copy_half_spinor<PREC, DAG ? 1 : 2>(STP + f * TM_HALF_TILE + sl, tp + f * STB, l);
            tile_copy_half_spinor<PREC, DAG ? 2 : 1>(STM + f * TM_HALF_TILE + sl, tmn + f * STB, l);
        }
        tile_copy_link<PREC, RECON>(LBT + sl, link_tile(gb_l, Ttm, 3), l);
    }
    cp_async_commit();

    // hop weights (HopCtx of tm_dslash_f2.cuh): time boundary sign, and 0 for a hop that leaves a cut sub-lattice
    HopCtx c;
    c.site = T * TM_TILE + l;
    c.wt[0] = 2.f * ((t == a.T - 1) ? (float)a.tbound : 1.f);
    c.wt[1] = 2.f * ((t == 0) ? (float)a.tbound : 1.f);
    c.ws[0] = (y == a.Y - 1) ? a.wrap_y : 1.f;
    c.ws[1] = (y == 0) ? a.wrap_y : 1.f;
    c.ws[2] = (z == a.Z - 1) ? a.wrap_z : 1.f;
    c.ws[3] = (z == 0) ? a.wrap_z : 1.f;

    f2 A[NF * 12], X[NF * 12];
#pragma unroll
    for (int i = 0; i < NF * 12; i++) A[i] = mk2(0.f, 0.f);
    HopRaw<PREC, NF, RECON> r;
    const int xp = q ? ((xh == Xh - 1) ? l - (Xh - 1) : l + 1) : l;          // x: the neighbours are in the tile of the same index
    const int xm = q ? l : ((xh == 0) ? l + (Xh - 1) : l - 1);
    const bool up_own = row < R - 1, dn_own = row > 0;                       // y: one row up / down inside the tile, or the y-tile
    const int yp = up_own ? l + Xh : xh, ym = dn_own ? l - Xh : 32 - Xh + xh;
    const unsigned SYP = up_own ? SX : SY, SYM = dn_own ? SX : SY;

    // ---- 2. the hops, from shared memory
    cp_async_wait<3>();
    __syncwarp();
    tile_read_hop<PREC, NF, RECON, 0>(r, SX, LF, xp, l);
    consume_hop<PREC, NF, RECON, DAG, false, 0>(A, r, c);
    tile_read_hop<PREC, NF, RECON, 0>(r, SX, LBX, xm, xm);
    consume_hop<PREC, NF, RECON, DAG, false, 1>(A, r, c);
    cp_async_wait<2>();
    __syncwarp();
    tile_read_hop<PREC, NF, RECON, 0>(r, SYP, LF + LTB, yp, l);
    consume_hop<PREC, NF, RECON, DAG, false, 2>(A, r, c);
    tile_read_hop<PREC, NF, RECON, 0>(r, SYM, LBY, ym, ym);
    consume_hop<PREC, NF, RECON, DAG, false, 3>(A, r, c);
    if constexpr (KT != 0) {
        // the x operand of the epilogue (the warp's own tile of another field) takes the place of the own-index tile, which the x and y hops
        // are done with: a fifth commit group, in flight during the z and t hops
        __syncwarp();
        const char *x_l = static_cast<const char *>(a.x) + l * 16;
        const char *xs = x_l + (size_t)(unsigned)T * FS;
#pragma unroll
        for (int f = 0; f < NF; f++) tile_copy_spinor<PREC, 0>(SX + f * STB + sl, xs + f * STB, l);
        cp_async_commit();
    }
    cp_async_wait<(KT != 0) ? 2 : 1>();
    __syncwarp();
    tile_read_hop<PREC, NF, RECON, 0>(r, SZP, LF + 2 * LTB, l, l);
    consume_hop<PREC, NF, RECON, DAG, false, 4>(A, r, c);
    tile_read_hop<PREC, NF, RECON, 0>(r, SZM, LBZ, l, l);
    consume_hop<PREC, NF, RECON, DAG, false, 5>(A, r, c);
    cp_async_wait<(KT != 0) ? 1 : 0>();
    __syncwarp();
    tile_read_hop<PREC, NF, RECON, DAG ? 1 : 2>(r, STP, LF + 3 * LTB, l, l);
    consume_hop<PREC, NF, RECON, DAG, false, 6>(A, r, c);
    tile_read_hop<PREC, NF, RECON, DAG ? 2 : 1>(r, STM, LBT, l, l);
    consume_hop<PREC, NF, RECON, DAG, false, 7>(A, r, c);

    // a7, a8: the epilogue and the single store of tm_dslash_f2 (x and out are the warp's own tile: one address)
    if constexpr (KT != 0) {
        cp_async_wait<0>();
        __syncwarp();
        tile_read_spinor<PREC, NF, RECON>(r, SX, l);
        load_x<PREC, NF, RECON>(X, r);
    }
    epilogue_f2<NF, KT>(A, X, (float)a.alpha, (float)a.beta, (float)a.scale, (float)a.kappa, (float)a.kappa2);
    char *os = static_cast<char *>(a.out) + (size_t)T * FS + (size_t)l * 16;
#pragma unroll
    for (int f = 0; f < NF; f++) store_spinor_f2<PREC>(A + 12 * f, os + f * STB, l);
}

template <int PREC, int NF, int RECON, int KT, bool DAG>
cudaError_t tm_launch_tile(const DslashArgs &a, cudaStream_t s)
{
    TileGeom tg;
    tg.Xh = a.Xh;
    tg.R = 32 / a.Xh;
    tg.tps = a.Y / tg.R;
    tg.lg = a.Xh == 4 ? 2 : a.Xh == 8 ? 3 : 4;
    tg.dtps = tm_fastdiv(tg.tps > 1 ? tg.tps : 2);       // not used when tps == 1
    tg.dZ = tm_fastdiv(a.Z);
    const size_t PB = (size_t)tm_tiles(a.Vh) * 4 * link_tile_bytes(PREC, RECON);
    tg.gauge_f = static_cast<const char *>(a.gauge) + (size_t)a.parity * PB;
    tg.gauge_b = static_cast<const char *>(a.gauge) + (size_t)(1 - a.parity) * PB;
    const size_t smem = (size_t)NF * (4 * spinor_tile_bytes(PREC) + 2 * TM_HALF_TILE) + (size_t)8 * link_tile_bytes(PREC, RECON);
    static std::atomic<unsigned long long> raised{0};
    cudaError_t e = tm_raise_smem(tm_dslash_tile<PREC, NF, RECON, KT, DAG>, raised);
    if (e != cudaSuccess) return e;
    return tm_launch_kernel(tm_dslash_tile<PREC, NF, RECON, KT, DAG>, a.pdl, a.Vh / TM_TILE, 32, smem, s, a, tg);
}
// the lattices the tile kernel covers (tm_dslash_apply falls back to the thread-per-site kernels otherwise)
inline bool tm_tile_geometry_ok(int Xh, int Y, int Vh) { return (Xh == 4 || Xh == 8 || Xh == 16) && Y % (32 / Xh) == 0 && Vh % TM_TILE == 0; }

// table index: [recon18 ? 0 : 1][kt 0..3][dagger 0..1]
#define TM_TILE_ROW(P, N, R, K)                                                          \
    {tm_launch_tile<P, N, R, K, false>, "tile<" #P "," #N "," #R "," #K ",plain>"},     \
    {tm_launch_tile<P, N, R, K, true>, "tile<" #P "," #N "," #R "," #K ",dagger>"}
#define TM_TILE_TABLE(P, N)                                                                                                  \
    static const TmKernelEntry tile_table_##P##_##N[16] = {TM_TILE_ROW(P, N, 18, 0), TM_TILE_ROW(P, N, 18, 1), TM_TILE_ROW(P, N, 18, 2), \
                                                           TM_TILE_ROW(P, N, 18, 3), TM_TILE_ROW(P, N, 12, 0), TM_TILE_ROW(P, N, 12, 1), \
                                                           TM_TILE_ROW(P, N, 12, 2), TM_TILE_ROW(P, N, 12, 3)};               \
    const TmKernelEntry *tm_tile_table_##P##_##N() { return tile_table_##P##_##N; }

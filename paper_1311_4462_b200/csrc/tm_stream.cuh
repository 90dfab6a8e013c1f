// tm_stream.cuh -- keeping HBM streaming ahead of the compute: L2 prefetch of a later tile.
//
// The gauge field is read exactly once per dslash (8 links per output site, no reuse) and is 2/3 of the HBM
// traffic; the input spinor is first touched by the forward-time hop of the site one time-slice below it.
// Both are plain contiguous segments per plane for a block of consecutive checkerboard sites, so the block
// with index b issues one cp.async.bulk.prefetch.L2 per segment for the sites of block b + pf_dist.  The
// loads of that later block then hit the 126 MB L2 (latency roughly halved) and the amount of data in flight
// from HBM no longer depends on how many registers a thread can spare for outstanding loads.
// Prefetches are hints: ranges are clamped / rounded, wraps are approximated, correctness never depends on them.
#pragma once
#include "tm_internal.h"
#include "tm_layout.cuh"

template <int PREC, int NF, int RECON, bool HAS_X>
TM_DEV void prefetch_tile(const DslashArgs &a, int sites_per_block, int vblock)
{
    if (a.pf_dist <= 0) return;
    const int Vh = a.Vh;
    const long first_l = (long)(vblock + a.pf_dist) * sites_per_block;
    if (first_l >= Vh) return;
    const int first = (int)first_l;
    const int n = min(sites_per_block, Vh - first);
    constexpr int NP = link_planes<PREC, RECON>();
    constexpr int NCH = PrecTraits<PREC>::NCH;
    constexpr int NSP = NF * (NCH + (PREC == 2 ? 1 : 0));          // spinor planes (+ norm plane in half)
    constexpr int NSEG = 8 * NP + NSP * (HAS_X ? 2 : 1);
    const size_t blk = (size_t)RECON * PREC * Vh;
    const int st = a.Xh * a.Y * a.Z;
    const size_t fl_bytes = (size_t)NCH * Vh * 16;
    for (int s = threadIdx.x; s < NSEG; s += blockDim.x) {
        if (s < 8 * NP) {
            const int dir = s / NP, plane = s - dir * NP, mu = dir & 3;
            const bool fwd = dir < 4;
            const int w = link_plane_width<PREC, RECON>(plane);
            int idx = first, cnt = n;
            if (!fwd) {                                              // U_mu(x - mu) lives at the neighbour's index
                idx = first - (mu == 0 ? 0 : mu == 1 ? a.Xh : mu == 2 ? a.Xh * a.Y : st);
                if (idx < 0) idx += Vh;
                idx &= ~3;
                cnt = min(n, Vh - idx);
            }
            const char *base = static_cast<const char *>(a.gauge) + (size_t)(fwd ? a.parity : 1 - a.parity) * 4 * blk +
                               (size_t)mu * blk + (size_t)link_plane_offset<PREC, RECON>(plane) * Vh;
            prefetch_l2(base + (size_t)idx * w, (unsigned)(cnt * w));
        } else {
            int r = s - 8 * NP;
            const bool isx = r >= NSP;
            if (isx) r -= NSP;
            const char *fb = static_cast<const char *>(isx ? a.x : a.in);
            int idx = first;
            if (!isx) {                                              // first touch: the forward time hop
                idx = first + st;
                if (idx >= Vh) idx -= Vh;
            }
            const int cnt = min(n, Vh - idx);
            const int f = r / (NSP / NF), k = r % (NSP / NF);
            if (k < NCH) prefetch_l2(fb + f * fl_bytes + ((size_t)k * Vh + idx) * 16, (unsigned)(cnt * 16));
            else prefetch_l2(fb + NF * fl_bytes + ((size_t)f * Vh + idx) * 4, (unsigned)(cnt * 4));
        }
    }
}

// ---- staging the link stream through shared memory with cp.async (LDGSTS) ------------------------------------
// Every thread starts the copy of all 8 links of its site before it does anything else, one commit group per hop,
// into [hop][plane][thread] slots (16-byte slots of consecutive threads are consecutive: conflict-free LDS.128).
// The bytes are then in flight without holding registers; hop h waits for group h only (cp.async.wait_group 7-h).
// A thread reads back only what it copied itself, so no block barrier is needed.
TM_DEV unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
template <int W> TM_DEV void cp_async(void *smem, const void *g)
{
    if constexpr (W == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem)), "l"(g) : "memory");
    else if constexpr (W == 8) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(smem)), "l"(g) : "memory");
    else asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(smem)), "l"(g) : "memory");
}
TM_DEV void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> TM_DEV void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <int PREC, int RECON>
TM_DEV void stage_link_nc(char *sm_hop, const char *gauge_blk, int Vh, int idx, int nt, int tid)     // no commit
{
    constexpr int NP = link_planes<PREC, RECON>();
#pragma unroll
    for (int p = 0; p < NP; p++) {
        const int w = link_plane_width<PREC, RECON>(p), o = link_plane_offset<PREC, RECON>(p);
        char *dst = sm_hop + (size_t)o * nt + (size_t)tid * w;
        const char *src = gauge_blk + (size_t)o * Vh + (size_t)idx * w;
        if (w == 16) cp_async<16>(dst, src);
        else if (w == 8) cp_async<8>(dst, src);
        else cp_async<4>(dst, src);
    }
}
template <int PREC, int RECON>
TM_DEV void stage_link(char *sm_hop, const char *gauge_blk, int Vh, int idx, int nt, int tid)
{
    stage_link_nc<PREC, RECON>(sm_hop, gauge_blk, Vh, idx, nt, tid);
    cp_async_commit();
}

// Where hop h finds its link: the staged [plane][thread] slots of the block, or the gauge block in global memory.
extern __shared__ __align__(16) char tm_smem[];
struct LinkSrc {
    const char *base;
    int stride;     // sites per plane
    int idx;
};
template <bool STG> TM_DEV LinkSrc link_src(int h, int link_bytes, const char *gauge_blk, int Vh, int gidx)
{
    LinkSrc L;
    if constexpr (STG) {
        L.base = tm_smem + (size_t)h * link_bytes * blockDim.x;
        L.stride = blockDim.x;
        L.idx = threadIdx.x;
    } else {
        L.base = gauge_blk;
        L.stride = Vh;
        L.idx = gidx;
    }
    return L;
}

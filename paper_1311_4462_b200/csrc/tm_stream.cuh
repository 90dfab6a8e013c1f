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

// Programmatic dependent launch (tm_launch_kernel, tm_internal.h).  tm_pdl_enter() is the first statement of every fused kernel: with the
// launch attribute the kernel may be set up on the GPU while the previous kernel of the stream is still running, and this instruction
// then holds it until that kernel has completed and its writes are visible -- before any field is read or written.  No kernel signals
// griddepcontrol.launch_dependents early (measured: blocks of the next kernel resident during the last wave make the step 25 % slower,
// profiles/r2_tuning.md section 10), so the order of execution is that of plain launches; what is saved is the launch gap (1.1 % of the
// step).  A no-op in a kernel launched without the attribute.
TM_DEV void tm_pdl_enter()
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

template <int PREC, int NF, int RECON, bool HAS_X>
TM_DEV void prefetch_tile(const DslashArgs &a, int sites_per_block, int vblock)
{
    if (a.pf_dist <= 0) return;
    const int Vh = a.Vh;
    const long first_l = (long)(vblock + a.pf_dist) * sites_per_block;      // a multiple of TM_TILE
    if (first_l >= Vh) return;
    const int first = (int)first_l;
    const int tiles = tm_tiles(Vh);
    const int t0 = first >> TM_TILE_LOG;
    const int nt = min((sites_per_block + TM_TILE - 1) >> TM_TILE_LOG, tiles - t0);
    constexpr int STB = NF * spinor_tile_bytes(PREC);
    constexpr int LTB = link_tile_bytes(PREC, RECON);
    const size_t PB = (size_t)tiles * 4 * LTB;                               // one parity's gauge block
    const int st = a.Xh * a.Y * a.Z;
    const int nseg = 3 + 4 * (nt + 1);
    for (int s = threadIdx.x; s < nseg; s += blockDim.x) {
        if (s == 0) {                                    // forward links: the block's own tiles, all four mu
            prefetch_l2(static_cast<const char *>(a.gauge) + (size_t)a.parity * PB + (size_t)t0 * 4 * LTB, (unsigned)(nt * 4 * LTB));
        } else if (s == 1) {                             // input spinor: first touched by the forward time hop
            int idx = first + st;
            if (idx >= Vh) idx -= Vh;
            const int ti = idx >> TM_TILE_LOG;
            prefetch_l2(static_cast<const char *>(a.in) + (size_t)ti * STB, (unsigned)(min(nt + 1, tiles - ti) * STB));
        } else if (s == 2) {
            if (HAS_X) prefetch_l2(static_cast<const char *>(a.x) + (size_t)t0 * STB, (unsigned)(nt * STB));
        } else {                                         // backward links U_mu(x - mu): the neighbour's tiles, one mu each
            const int r = s - 3, mu = r & 3, j = r >> 2;
            int idx = first - (mu == 0 ? 0 : mu == 1 ? a.Xh : mu == 2 ? a.Xh * a.Y : st);
            if (idx < 0) idx += Vh;
            const int tb = (idx >> TM_TILE_LOG) + j;
            if (tb < tiles)
                prefetch_l2(static_cast<const char *>(a.gauge) + (size_t)(1 - a.parity) * PB + ((size_t)tb * 4 + mu) * LTB, (unsigned)LTB);
        }
    }
}

// ---- staging the link stream through shared memory with cp.async (LDGSTS) ------------------------------------
// Every thread starts the copy of all 8 links of its site before it does anything else, one commit group per hop,
// into the slot [hop][warp] of RECON * PREC * 32 bytes that has the tile shape [plane][32 lanes] (conflict-free
// LDS.128, and load_link reads it with the same offsets as a tile in global memory).
// The bytes are then in flight without holding registers; hop h waits for group h only (cp.async.wait_group 7-h).
// A thread reads back only what it copied itself, so no block barrier is needed.
TM_DEV unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
template <int W> TM_DEV void cp_async(void *smem, const void *g)
{
    if constexpr (W == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem)), "l"(g) : "memory");
    else if constexpr (W == 8) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(smem)), "l"(g) : "memory");
    else asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(smem)), "l"(g) : "memory");
}
// the same with the shared address as a 32-bit word (tm_dslash_tile.cuh)
template <int W> TM_DEV void cp_async_u32(unsigned smem, const void *g)
{
    if constexpr (W == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem), "l"(g) : "memory");
    else if constexpr (W == 8) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem), "l"(g) : "memory");
    else asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem), "l"(g) : "memory");
}
TM_DEV void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> TM_DEV void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

extern __shared__ __align__(16) char tm_smem[];
// the thread's pointer into the staged copy of hop h (plays the role of the link's site pointer)
template <int PREC, int RECON> TM_DEV char *stage_slot(int h)
{
    const int warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5, lane = threadIdx.x & 31;
    return tm_smem + (size_t)(h * nwarps + warp) * link_tile_bytes(PREC, RECON) + lane * 16;
}
template <int PREC, int RECON>
TM_DEV void stage_link(int h, const char *lp, int src_lane)      // src_lane = (index of the link's site) & 31
{
    constexpr int N16 = link_n16<PREC, RECON>(), TW = link_tailw<PREC, RECON>();
    const int lane = threadIdx.x & 31;
    char *dst = stage_slot<PREC, RECON>(h);
#pragma unroll
    for (int k = 0; k < N16; k++) cp_async<16>(dst + k * TM_PLANE, lp + k * TM_PLANE);
    if constexpr (TW == 8) cp_async<8>(dst + tail_off(N16, 8, lane), lp + tail_off(N16, 8, src_lane));
    if constexpr (TW == 4) cp_async<4>(dst + tail_off(N16, 4, lane), lp + tail_off(N16, 4, src_lane));
    cp_async_commit();
}

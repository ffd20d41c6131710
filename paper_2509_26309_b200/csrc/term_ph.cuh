// term_ph.cuh -- the hot kernel: fused Chebyshev term, TMA-staged MATRIX slices, directly streamed VECTORS, and an
// explicitly phased instruction stream (all index loads -> all global loads -> all complex FMAs).
//
//   T_k = a*H*T_{k-1} - T_{k-2}  (amxsy)  fused with  psi' += sum c_j T_j  (axpy, up to
//   three terms at once) and, on the last term of a time step, <psi0|psi'> and <psi'|psi'> (calc_corr_dos).
//
// Why this shape (profiles/r1b_ncu_full_cfg2-5.md): with 8 interleaved states per row the previous kernel (term_ws.cu)
// was bound in the SM clock domain -- by L1 data-pipe wavefronts (16-25 per row where the gathers and the store need
// 8-10) and by three to four serialised memory round trips per row (a warp pass took ~4800 cycles).  Here
//   producer warp (one elected lane): for every tile of R rows, n_stage tiles ahead, bulk-copies (cp.async.bulk +
//       mbarrier complete_tx; SASS UBLKCP) ONLY the matrix slices of the tile -- row offsets, packed column words,
//       value indices (large tables only), real diagonal -- into a 2-7 KB shared-memory stage;
//   consumer warps: issue the streamed operands of their row (y, psi', psi0, x[row]; coalesced 128/256-bit LDG) before
//       they even wait for the stage; then read ALL their indices from shared memory, release the stage at once
//       (the producer refills it while the gathers are in flight), issue ALL gathers of x[col] back to back (one
//       memory round trip per row of <= CH entries), and only then run the complex FMAs.  Results go straight to
//       global memory.  No block-wide barrier in the main loop.
//
// Thread -> (row, SPT consecutive states).  What varies per term (accumulate 0..3 terms, reduce or not) is a template
// parameter; what varies rarely (first term, first flush, diagonal present) is a warp-uniform runtime predicate.
#pragma once

#include <algorithm>

#include "ptx_helpers.cuh"
#include "term.h"

namespace tbpm_detail {
namespace ph {

constexpr int kMaxStages = 8;
constexpr int kNwA = 23, kNwB = 19;       // consumer warps of the short-row / six-entry shapes (see launch_bt)

using namespace ptx;

// SPT consecutive complex128 values of one row
template <int SPT> struct CVec;
template <> struct CVec<1> {
    double2 v[1];
    __device__ __forceinline__ void zero() { v[0] = make_double2(0.0, 0.0); }
    __device__ __forceinline__ void gather_if(const double2 *p, bool on)      // read-only path, cacheable; zeros when off
    {
        asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %3, 0;\nmov.f64 %0, 0d0000000000000000;\nmov.f64 %1, 0d0000000000000000;\n"
                     "@q ld.global.nc.v2.f64 {%0, %1}, [%2];\n}"
                     : "=d"(v[0].x), "=d"(v[0].y)
                     : "l"(p), "r"((int)on));
    }
    __device__ __forceinline__ void gather(const double2 *p)
    {
        asm volatile("ld.global.nc.v2.f64 {%0, %1}, [%2];" : "=d"(v[0].x), "=d"(v[0].y) : "l"(p));
    }
    __device__ __forceinline__ void stream_if(const double2 *p, bool on)      // read once: evict first
    {
        asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %3, 0;\nmov.f64 %0, 0d0000000000000000;\nmov.f64 %1, 0d0000000000000000;\n"
                     "@q ld.global.cs.v2.f64 {%0, %1}, [%2];\n}"
                     : "=d"(v[0].x), "=d"(v[0].y)
                     : "l"(p), "r"((int)on)
                     : "memory");
    }
    __device__ __forceinline__ void st(double2 *p) const
    {
        asm volatile("st.global.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(v[0].x), "d"(v[0].y) : "memory");
    }
    __device__ __forceinline__ void st_stream(double2 *p) const
    {
        asm volatile("st.global.cs.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(v[0].x), "d"(v[0].y) : "memory");
    }
};
template <> struct CVec<2> {
    double2 v[2];
    __device__ __forceinline__ void zero() { v[0] = v[1] = make_double2(0.0, 0.0); }
    __device__ __forceinline__ void gather_if(const double2 *p, bool on)      // one 256-bit load (LDG.E.256)
    {
        asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %5, 0;\nmov.f64 %0, 0d0000000000000000;\nmov.f64 %1, 0d0000000000000000;\n"
                     "mov.f64 %2, 0d0000000000000000;\nmov.f64 %3, 0d0000000000000000;\n"
                     "@q ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];\n}"
                     : "=d"(v[0].x), "=d"(v[0].y), "=d"(v[1].x), "=d"(v[1].y)
                     : "l"(p), "r"((int)on));
    }
    __device__ __forceinline__ void gather(const double2 *p)
    {
        asm volatile("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(v[0].x), "=d"(v[0].y), "=d"(v[1].x), "=d"(v[1].y) : "l"(p));
    }
    __device__ __forceinline__ void stream_if(const double2 *p, bool on)
    {
        asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %5, 0;\nmov.f64 %0, 0d0000000000000000;\nmov.f64 %1, 0d0000000000000000;\n"
                     "mov.f64 %2, 0d0000000000000000;\nmov.f64 %3, 0d0000000000000000;\n"
                     "@q ld.global.L1::no_allocate.L2::evict_first.v4.f64 {%0, %1, %2, %3}, [%4];\n}"
                     : "=d"(v[0].x), "=d"(v[0].y), "=d"(v[1].x), "=d"(v[1].y)
                     : "l"(p), "r"((int)on)
                     : "memory");
    }
    __device__ __forceinline__ void st(double2 *p) const
    {
        asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(v[0].x), "d"(v[0].y), "d"(v[1].x), "d"(v[1].y) : "memory");
    }
    __device__ __forceinline__ void st_stream(double2 *p) const
    {
        asm volatile("st.global.L1::no_allocate.L2::evict_first.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(v[0].x), "d"(v[0].y), "d"(v[1].x),
                     "d"(v[1].y)
                     : "memory");
    }
};

__device__ __forceinline__ double2 ldg_value_if(const double2 *p, bool on)
{
    double2 v;
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %3, 0;\nmov.f64 %0, 0d0000000000000000;\nmov.f64 %1, 0d0000000000000000;\n"
                 "@q ld.global.nc.v2.f64 {%0, %1}, [%2];\n}"
                 : "=d"(v.x), "=d"(v.y)
                 : "l"(p), "r"((int)on));
    return v;
}

// BT states per tile row, SPT states per thread, CH gathers in flight per thread, NACC terms added to psi' by this launch
// (0..3), REDUCE: last term of the time step (dot products, T_k not stored).
// VK, where the hopping values come from:  0 = 15-bit index + conjugate bit per entry into the table in global memory
//   (4 = the same with the table copied into shared memory);
//   1 = ONE value, in registers, v or conj(v) by bit 31 of the packed column word (build.cu);  2 = ONE REAL value (clean lattices,
//   Anderson disorder, vacancies): the neighbours are summed and the sum scaled once -- 2 DADD per entry and state
//   where the complex FMA takes 4 DFMA.
// UNI: every row holds exactly max_row_off entries, a multiple of CH (periodic lattices): no row offsets, no predicates.
// NW consumer warps + 1 producer warp form the only block of an SM: (NW + 1) * 32 threads share the 64 K registers.
template <int BT, int SPT, int CH, int NACC, bool REDUCE, int VK, bool UNI, int NW>
__global__ void __launch_bounds__((NW + 1) * 32, 1) k_term_ph(const TermParams p)
{
    constexpr int kConsumers = NW * 32;
    constexpr int LPR = BT / SPT;                           // lanes per row
    constexpr int R = kConsumers / LPR;                     // rows per tile
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t bars[2 * kMaxStages];  // [0, S): full, [kMaxStages, kMaxStages + S): empty
    __shared__ uint32_t lo_s[kMaxStages][2];                // first column / value-index element held by each stage
    __shared__ double red_s[REDUCE ? kConsumers / 32 : 1][REDUCE ? BT : 1][3];

    const int tid = threadIdx.x;
    const bool sub_y = p.flags & F_SUB_Y;
    const bool need_y = sub_y || NACC == 3;
    const bool need_acc = NACC > 0 && !(p.flags & F_ACC_INIT);
    const bool has_diag = p.diag != nullptr;
    const bool need_xrow = NACC >= 2 || has_diag;
    const int S = p.n_stage;
    const int64_t n_tiles = (p.n_orb + R - 1) / R;
    const uint32_t bar0 = smem_u32(bars), smem0 = smem_u32(smem);

    if (tid == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(bar0 + 8 * s, 1); mbar_init(bar0 + 8 * (kMaxStages + s), kConsumers / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (VK == 4) {                                          // the whole (conjugate-folded) value table, once per block
        double2 *tab = reinterpret_cast<double2 *>(smem + (size_t)p.stage_bytes * p.n_stage);
        for (int i = tid; i < p.n_table; i += (NW + 1) * 32) tab[i] = __ldg(p.vtab + i);
    }
    __syncthreads();

    // Tile order of a block.  The tiles are viewed as a [line][d0] grid (d0 tiles per lattice line; d0 = 1: no lattice
    // known) and dealt to the blocks in RUNS of `len` tiles that step one line at a time: run u covers the tiles
    // ((u / d0) * len + i) * d0 + u % d0, i < len.  Inside a run the rows gathered for one tile (the neighbours one line
    // up and down) are the rows of the run's previous and next tiles, so they are found in the SM's L1 instead of crossing
    // the L2 fabric again; all blocks together still sweep one moving window of the vectors (L2 locality).
    const int64_t d0 = p.walk_d0;
    const int wlen = p.walk_len;
    auto run_base = [&](int64_t u) -> int64_t {
        const int64_t lb = u / d0;
        const int64_t t = lb * wlen * d0 + (u - lb * d0);
        return t < n_tiles ? t : n_tiles;                   // the base grows with u: the first one past the end ends the walk
    };
    auto next_tile = [&](int64_t t, int &i, int64_t &u) -> int64_t {
        if (++i < wlen) { t += d0; if (t < n_tiles) return t; }
        i = 0;
        u += gridDim.x;
        return run_base(u);
    };
    const int64_t first_tile = run_base(blockIdx.x);
    // Every other term sweeps the rows from the end: what the previous term wrote and gathered last is still in L2 when this
    // term starts there (worth 20-25 % of the DRAM reads when the vectors are a few times the L2, nothing when far larger).
    const bool rev = p.reverse != 0;
    auto tile_rows = [&](int64_t t) -> int64_t { return (rev ? n_tiles - 1 - t : t) * R; };

    if (tid >= kConsumers) {
        // ------------------------------------------------ producer warp ------------------------------------------------
        // Lane 0 stages the matrix slices.  All 32 lanes then PREFETCH INTO L2 the vector rows that a tile `pf_dist` steps
        // further along this block's walk will stream (y, psi', psi0) or touch first (x at the leading edge of the gather
        // window): the consumers hold one row group per warp in registers, which keeps only ~30 KB of DRAM-bound loads
        // in flight per SM where the HBM needs ~64 KB (microbenchmark, profiles/r2_microbench.md); prefetches hold no
        // registers, so they carry the DRAM latency and the consumers' loads become L2 hits.
        const int lane = tid - kConsumers;
        uint32_t q_lo = 0, q_hi = 0;                        // offsets bounding the next tile to issue (prefetched)
        int64_t tile = first_tile;
        if (lane == 0 && tile < n_tiles) {
            const int64_t r0 = tile_rows(tile);
            q_lo = __ldg(p.orp + r0);
            q_hi = __ldg(p.orp + min(r0 + R, p.n_orb));
        }
        int s = 0, ci = 0;
        int64_t cu = blockIdx.x;
        uint32_t ph = 1;                                    // parity of the "empty" phase to wait for; first pass: free
        // cursor of the prefetched tile, pf_dist steps ahead of the staged one
        const int pfd = p.pf_dist;
        int64_t ptile = first_tile, pu = blockIdx.x;
        int pi = 0;
        for (int k = 0; k < pfd && ptile < n_tiles; ++k) ptile = next_tile(ptile, pi, pu);
        for (; tile < n_tiles; tile = next_tile(tile, ci, cu)) {
            if (lane == 0) {
                const uint32_t c_lo = q_lo, c_hi = q_hi;
                int cj = ci;
                int64_t cv = cu;
                const int64_t nt = next_tile(tile, cj, cv);
                if (nt < n_tiles) {                         // bounds of the following tile: latency hidden behind this issue
                    const int64_t nr0 = tile_rows(nt);
                    q_lo = __ldg(p.orp + nr0);
                    q_hi = __ldg(p.orp + min(nr0 + R, p.n_orb));
                }
                const uint32_t full = bar0 + 8 * s;
                mbar_wait(bar0 + 8 * (kMaxStages + s), ph); // a fresh barrier reports the "previous" phase complete
                const uint32_t st = smem0 + (uint32_t)s * (uint32_t)p.stage_bytes;
                const int64_t r0 = tile_rows(tile);
                const int rows = (int)min((int64_t)R, p.n_orb - r0);
                const uint32_t col_lo = c_lo & ~3u, idx_lo = c_lo & ~7u;
                const uint32_t nc = ((c_hi - col_lo) + 3u) & ~3u, ni = ((c_hi - idx_lo) + 7u) & ~7u;
                lo_s[s][0] = col_lo;
                lo_s[s][1] = idx_lo;
                const uint32_t orp_bytes = (uint32_t)(((rows + 1) * 4 + 15) & ~15);
                uint32_t tx = orp_bytes;
                bulk_g2s(st, p.orp + r0, orp_bytes, full);
                if (nc > 0) {
                    bulk_g2s(st + p.off_col, p.ocol + col_lo, nc * 4, full);
                    tx += nc * 4;
                    if (VK == 0 || VK == 4) { bulk_g2s(st + p.off_idx, p.oidx + idx_lo, ni * 2, full); tx += ni * 2; }
                }
                if (has_diag) {
                    const uint32_t db = (uint32_t)((rows * 8 + 15) & ~15);
                    bulk_g2s(st + p.off_diag, p.diag + r0, db, full);
                    tx += db;
                }
                mbar_expect_tx(full, tx);                   // release: also publishes lo_s[s]
                if (++s == S) { s = 0; ph ^= 1u; }
            }
            __syncwarp();                                   // the prefetches follow the pace of the stages
            if (pfd > 0 && ptile < n_tiles) {
                const int64_t r0 = tile_rows(ptile);
                const int64_t rows = min((int64_t)R, p.n_orb - r0);
                const int n_lines = (int)((rows * BT * 16 + 127) >> 7);
                const char *py = reinterpret_cast<const char *>(p.y + r0 * BT);
                const char *pa = reinterpret_cast<const char *>(p.acc + r0 * BT);
                const char *pz = reinterpret_cast<const char *>(p.psi0 + r0 * BT);
                const int64_t x0 = r0 + p.pf_lead;          // leading edge of the gather window of that tile
                const char *px = reinterpret_cast<const char *>(p.x + x0 * BT);
                const bool x_ok = x0 >= 0 && x0 + rows <= p.n_orb;
                const bool do_y = need_y && (p.pf_mask & 1), do_x = x_ok && (p.pf_mask & 2);
                for (int o = lane; o < n_lines; o += 32) {
                    if (do_y) prefetch_l2(py + (size_t)o * 128);
                    if (do_x) prefetch_l2(px + (size_t)o * 128);
                    if (NACC > 0 && need_acc) prefetch_l2(pa + (size_t)o * 128);
                    if (REDUCE) prefetch_l2(pz + (size_t)o * 128);
                }
                ptile = next_tile(ptile, pi, pu);
            }
        }
        return;
    }

    // ---------------------------------------------------- consumer warps ----------------------------------------------------
    const int rl = tid / LPR;                               // row within the tile
    const int b0 = (tid % LPR) * SPT;                       // first state of this thread
    const double2 *xb = p.x + b0;
    const bool st_ef = p.pol & 1;                           // T_k leaves L2 first (its readers come a whole sweep later)
    const uint32_t stage_bytes = (uint32_t)p.stage_bytes;
    const uint32_t n_uni = (uint32_t)p.max_row_off;         // UNI: every row holds exactly this many entries (a multiple of CH)
    const uint32_t tab0 = smem0 + (uint32_t)p.stage_bytes * (uint32_t)p.n_stage;   // VK 4: the value table behind the stages
    const uint32_t a_orp = smem0 + (uint32_t)rl * 4u, a_col = smem0 + (uint32_t)p.off_col, a_idx = smem0 + (uint32_t)p.off_idx,
                   a_diag = smem0 + (uint32_t)p.off_diag;
    double2 t0 = make_double2(0.0, 0.0), t1 = t0;           // VK >= 1: the one hopping value and its conjugate, in registers
    if (VK >= 1) {
        t0 = __ldg(p.vtab);
        t1 = make_double2(t0.x, -t0.y);                     // the one table value and its conjugate (bit 31 of the column word)
    }
    double s_re[SPT], s_im[SPT], s_nn[SPT];
#pragma unroll
    for (int k = 0; k < SPT; ++k) s_re[k] = s_im[k] = s_nn[k] = 0.0;

    // The loop is ROTATED: an iteration first consumes the chunk that the previous iteration (or the prologue) loaded,
    // then loads the next chunk.  The loads and their uses are thereby separated by the loop back edge, which the
    // assembler's scheduler does not move code across -- left in one basic block it sinks six of eight gathers below the
    // first complex FMA and serialises the memory round trips.
    int s = 0;
    uint32_t ph = 0, so = 0;                                // so: byte offset of stage s
    int64_t tile = first_tile, cu = blockIdx.x;
    int ci = 0;
    bool valid = false;
    int64_t e = 0;
    uint32_t n = 0, nmax = 0, c0 = 0, ca = 0, ia = 0;
    double d = 0.0;
    CVec<SPT> yold, xrow, aold, z, h;
    CVec<SPT> x[CH];
    double2 v[CH];
    uint32_t w[CH];
    uint32_t id[CH];                                        // VK 0/4: table index + conjugate bit of each entry of the chunk

    auto load_row = [&]() {                                 // streamed operands + row header of `tile`
        const int64_t trow = tile_rows(tile);
        const int64_t row = trow + rl;
        valid = row < p.n_orb;
        e = row * BT + b0;
        // streamed operands of the row (HBM latency; they need no index, so they leave before the wait)
        yold.stream_if(p.y + e, valid && need_y);
        if (NACC > 0) aold.stream_if(p.acc + e, valid && need_acc);
        if (REDUCE) z.stream_if(p.psi0 + e, valid);
        xrow.gather_if(p.x + e, valid && need_xrow);        // the tile's own x rows are gathered by its neighbours: L1/L2 hit
        mbar_wait(bar0 + 8 * s, ph);
        if (UNI) {                                          // rows past the end of the last tile redo its first row, unstored
            const uint32_t rle = valid ? (uint32_t)rl : 0u;
            const uint32_t q0 = (uint32_t)trow * n_uni;                // low 32 bits suffice for the offsets below
            n = nmax = n_uni;
            ca = a_col + so + (rle * n_uni + (q0 & 3u)) * 4u;
            ia = a_idx + so + (rle * n_uni + (q0 & 7u)) * 2u;
            d = has_diag ? lds_f64(a_diag + so + rle * 8u) : 0.0;
        } else {
            const uint32_t q0 = lds_u32(a_orp + so), q1 = lds_u32(a_orp + so + 4u);
            n = valid ? q1 - q0 : 0u;
            ca = a_col + so + (q0 - lo_s[s][0]) * 4u;
            ia = a_idx + so + (q0 - lo_s[s][1]) * 2u;
            d = has_diag ? lds_f64(a_diag + so + (uint32_t)rl * 8u) : 0.0;
            nmax = __reduce_max_sync(0xffffffffu, n);
        }
        c0 = 0;
        h.zero();
    };
    auto load_chunk = [&]() {                               // indices of entries [c0, c0 + CH) of the row, then their gathers
        if constexpr (UNI && CH % 4 == 0) {                 // uniform rows of 4k entries: the slices are 16-byte aligned
#pragma unroll
            for (int j = 0; j < CH; j += 4) {
                lds_v4_u32(ca + 4u * (c0 + j), w[j], w[j + 1], w[j + 2], w[j + 3]);
                if (VK == 0 || VK == 4) {
                    uint32_t lo, hi;
                    lds_v2_u32(ia + 2u * (c0 + j), lo, hi);
                    id[j] = lo & 0xffffu; id[j + 1] = lo >> 16; id[j + 2] = hi & 0xffffu; id[j + 3] = hi >> 16;
                } else {
                    id[j] = id[j + 1] = id[j + 2] = id[j + 3] = 0u;
                }
            }
        } else if constexpr (UNI && CH % 2 == 0 && VK != 0) { // uniform rows of 2k entries (cubic: 6): 8-byte aligned
#pragma unroll
            for (int j = 0; j < CH; j += 2) {
                lds_v2_u32(ca + 4u * (c0 + j), w[j], w[j + 1]);
                id[j] = id[j + 1] = 0u;
            }
        } else {
#pragma unroll
            for (int j = 0; j < CH; ++j) {
                if (UNI) {
                    w[j] = lds_u32(ca + 4u * (c0 + j));
                    id[j] = (VK == 0 || VK == 4) ? lds_u16(ia + 2u * (c0 + j)) : 0u;
                } else {
                    w[j] = lds_u32_if(ca + 4u * (c0 + j), c0 + j < n);
                    id[j] = (VK == 0 || VK == 4) ? lds_u16_if(ia + 2u * (c0 + j), c0 + j < n) : 0u;
                }
            }
        }
        if (c0 + CH >= nmax) {                              // last chunk of every row of this warp: the stage is free again
            // ... once its reads have RETURNED: the barrier address depends on every register they filled (p.zero is 0 at run time)
            uint32_t rel = (uint32_t)__double2hiint(d);
#pragma unroll
            for (int j = 0; j < CH; ++j) rel ^= w[j] ^ id[j];
            rel &= (uint32_t)p.zero;
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(bar0 + 8 * (kMaxStages + s) + rel);
            if (++s == S) { s = 0; ph ^= 1u; so = 0; } else so += stage_bytes;
        }
#pragma unroll
        for (int j = 0; j < CH; ++j) {
            const double2 *src = xb + (int64_t)(w[j] & 0x7fffffffu) * BT;
            if (UNI) x[j].gather(src); else x[j].gather_if(src, c0 + j < n);
        }
        if (VK == 0) {
#pragma unroll
            for (int j = 0; j < CH; ++j) v[j] = table_value(ldg_value_if(p.vtab + (id[j] & 0x7fffu), UNI || c0 + j < n), id[j]);
        }
    };

    if (tile < n_tiles) {
        load_row();
        load_chunk();
    }
#pragma unroll 1
    while (tile < n_tiles) {
        // ---- consume the chunk in flight, in issue order
        if (VK == 2) {                                      // one real hopping value: sum the neighbours, scale once per row
#pragma unroll
            for (int j = 0; j < CH; ++j) {
#pragma unroll
                for (int k = 0; k < SPT; ++k) { h.v[k].x += x[j].v[k].x; h.v[k].y += x[j].v[k].y; }   // x[j] is zero past the row end
            }
        } else {
            if (VK == 4) {                                  // values from the table in shared memory, only now: 30-cycle loads,
#pragma unroll                                               // no registers held for them while the gathers are in flight
                for (int j = 0; j < CH; ++j) {
                    double2 t;
                    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(t.x), "=d"(t.y) : "r"(tab0 + (id[j] & 0x7fffu) * 16u));
                    v[j] = table_value(t, id[j]);
                }
            }
#pragma unroll
            for (int j = 0; j < CH; ++j) {
                if (VK == 1) v[j] = (w[j] >> 31) ? t1 : t0;
#pragma unroll
                for (int k = 0; k < SPT; ++k) cfma(h.v[k], v[j], x[j].v[k]);
            }
        }
        c0 += CH;
        if (c0 >= nmax) {
            // ---- epilogue of the row: diagonal, scale, subtract, store, accumulate, reduce
            if (VK == 2) {
#pragma unroll
                for (int k = 0; k < SPT; ++k) { h.v[k].x *= t0.x; h.v[k].y *= t0.x; }
            }
            if (has_diag) {
#pragma unroll
                for (int k = 0; k < SPT; ++k) { h.v[k].x = fma(d, xrow.v[k].x, h.v[k].x); h.v[k].y = fma(d, xrow.v[k].y, h.v[k].y); }
            }
#pragma unroll
            for (int k = 0; k < SPT; ++k) { h.v[k].x *= p.a; h.v[k].y *= p.a; }
            if (sub_y) {
#pragma unroll
                for (int k = 0; k < SPT; ++k) { h.v[k].x -= yold.v[k].x; h.v[k].y -= yold.v[k].y; }
            }
            if (valid) {
                if (!REDUCE) { if (st_ef) h.st_stream(p.y + e); else h.st(p.y + e); }   // T_k
                if (NACC > 0) {
#pragma unroll
                    for (int k = 0; k < SPT; ++k) {
                        cfma(aold.v[k], p.ca, h.v[k]);
                        if (NACC >= 2) cfma(aold.v[k], p.cb, xrow.v[k]);
                        if (NACC == 3) cfma(aold.v[k], p.cc, yold.v[k]);
                    }
                    if (REDUCE) {
#pragma unroll
                        for (int k = 0; k < SPT; ++k) {
                            s_re[k] = fma(z.v[k].x, aold.v[k].x, s_re[k]);      // conj(z) * psi'
                            s_re[k] = fma(z.v[k].y, aold.v[k].y, s_re[k]);
                            s_im[k] = fma(z.v[k].x, aold.v[k].y, s_im[k]);
                            s_im[k] = fma(-z.v[k].y, aold.v[k].x, s_im[k]);
                            s_nn[k] = fma(aold.v[k].x, aold.v[k].x, s_nn[k]);
                            s_nn[k] = fma(aold.v[k].y, aold.v[k].y, s_nn[k]);
                        }
                        aold.st(p.acc + e);                 // psi': T_0 of the next step, gathered right away
                    } else {
                        aold.st_stream(p.acc + e);
                    }
                }
            }
            tile = next_tile(tile, ci, cu);
            if (tile >= n_tiles) break;
            load_row();
        }
        // ---- load: the next chunk (of this row, or the first of the next tile's row)
        load_chunk();
    }

    if (REDUCE) {
#pragma unroll
        for (int k = 0; k < SPT; ++k) {                     // lanes with equal (lane % LPR) hold the same states
#pragma unroll
            for (int o = 16; o >= LPR; o >>= 1) {
                s_re[k] += __shfl_xor_sync(0xffffffffu, s_re[k], o);
                s_im[k] += __shfl_xor_sync(0xffffffffu, s_im[k], o);
                s_nn[k] += __shfl_xor_sync(0xffffffffu, s_nn[k], o);
            }
        }
        const int lane = tid & 31, warp = tid >> 5;
        if (lane < LPR) {
#pragma unroll
            for (int k = 0; k < SPT; ++k) {
                red_s[warp][lane * SPT + k][0] = s_re[k];
                red_s[warp][lane * SPT + k][1] = s_im[k];
                red_s[warp][lane * SPT + k][2] = s_nn[k];
            }
        }
        asm volatile("bar.sync 1, %0;" ::"n"(kConsumers) : "memory");   // consumers only (the producer warp has left)
        if (tid < BT * 3) {
            const int bb = tid / 3, c = tid % 3;
            double t = 0.0;
#pragma unroll
            for (int w = 0; w < kConsumers / 32; ++w) t += red_s[w][bb][c];
            p.partial[((int64_t)blockIdx.x * BT + bb) * 3 + c] = t;
        }
    }
}

template <int BT, int SPT, int CH, int NACC, bool REDUCE, int VK, bool UNI, int NW>
int launch_one(TermParams p, int num_sms, cudaStream_t st, int *grid_out)
{
    constexpr int kConsumers = NW * 32, kThreads = kConsumers + 32;
    constexpr int R = kConsumers / (BT / SPT);
    p.n_stage = std::min(kMaxStages, std::max(2, knob("stages", 4)));
    p.walk_d0 = 1;
    p.walk_len = std::max(1, knob("chunk", 1));
    if (p.walk_stride > 0 && p.walk_stride % R == 0) {      // a lattice line is a whole number of tiles: walk across lines
        p.walk_d0 = p.walk_stride / R;
        p.walk_len = std::max(1, p.walk_run);
    }
    p.pol = knob("pol", 1);
    const StageGeom g = stage_geom(R, p.max_row_off, VK == 0 || VK == 4);
    p.cap_entries = g.cap_entries; p.off_col = g.off_col; p.off_idx = g.off_idx; p.off_diag = g.off_diag; p.off_vec = 0;
    p.stage_bytes = g.stage_bytes;
    const size_t tab = VK == 4 ? (size_t)p.n_table * sizeof(double2) : 0;
    const size_t room = std::min<size_t>(kStageBudget, kSmemMax - tab);
    if ((size_t)p.stage_bytes * 2 > room) return TBPM_EINVAL;   // term_ph_supported / launch_bt rule this out
    p.n_stage = (int)std::min<size_t>(p.n_stage, room / p.stage_bytes);
    const size_t dyn = (size_t)p.stage_bytes * p.n_stage + tab;
    auto kern = k_term_ph<BT, SPT, CH, NACC, REDUCE, VK, UNI, NW>;
    static size_t configured[kMaxDevices] = {0};            // per device: the attribute belongs to the device's copy of the function
    if (p.device < 0 || p.device >= kMaxDevices) return TBPM_EINVAL;
    if (dyn > configured[p.device]) {
        const size_t want = std::max(dyn, (size_t)64 * 1024);
        TBPM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)want));
        configured[p.device] = want;
    }
    const int64_t need = (p.n_orb + R - 1) / R;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>({need, (int64_t)num_sms, (int64_t)kMaxGrid}));   // one block per SM
    kern<<<grid, kThreads, dyn, st>>>(p);
    count_launches(1);
    *grid_out = grid;
    return TBPM_OK;
}

template <int BT, int SPT, int CH, int VK, bool UNI, int NW>
int launch_variant(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    const bool red = p.flags & F_REDUCE;
    if (!red && p.n_acc == 0) return launch_one<BT, SPT, CH, 0, false, VK, UNI, NW>(p, num_sms, st, grid_out);
    if (!red && p.n_acc == 3) return launch_one<BT, SPT, CH, 3, false, VK, UNI, NW>(p, num_sms, st, grid_out);
    if (red && p.n_acc == 1) return launch_one<BT, SPT, CH, 1, true, VK, UNI, NW>(p, num_sms, st, grid_out);
    if (red && p.n_acc == 2) return launch_one<BT, SPT, CH, 2, true, VK, UNI, NW>(p, num_sms, st, grid_out);
    if (red && p.n_acc == 3) return launch_one<BT, SPT, CH, 3, true, VK, UNI, NW>(p, num_sms, st, grid_out);
    return TBPM_EINVAL;
}

// Shape of the instruction stream, chosen from what the builder found (table size, one real value, uniform rows) and
// the tile width.  NW = 31 leaves 64 registers per thread, NW = 23 -> 80, NW = 19 -> 96, NW = 15 -> 128.
template <int BT>
int launch_bt(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    constexpr int SPT = BT >= 2 ? 2 : 1;
    const int n = p.max_row_off;
    const bool uni = p.uniform && knob("uni", 1);
    const int vk = (p.single_real && knob("vk2", 1)) ? 2 : (p.packed ? 1 : 0);
    if (uni && vk == 2 && n == 6) {
        // Three-dimensional lattice: walk the tiles along the largest stride (the plane).  A run then re-uses the rows it
        // gathered one plane down as its own rows and as the plane-up neighbours of its next tiles (L1), and the window
        // of T_{k-1} that must survive in L2 shrinks from two planes to the band the blocks work on -- the flush
        // launches stop re-reading it (ncu: 9.7 -> 7.1 GB per launch on cfg5).  16 consumer warps: 2^k rows per tile.
        TermParams q = p;
        constexpr int R16 = 512 / (BT / SPT);
        if (q.walk_stride == 0 && knob("autowalk", 1))
            for (int j = 0; j < q.n_lat_off; ++j)
                if (q.lat_off[j] % R16 == 0 && q.lat_off[j] * 4 <= q.n_orb) { q.walk_stride = q.lat_off[j]; q.walk_run = 64; }
        if (q.walk_stride > 0 && q.walk_stride % R16 == 0) return launch_variant<BT, SPT, 6, 2, true, 16>(q, num_sms, st, grid_out);
    }
    if constexpr (BT == 1) if (p.n_orb >= (int64_t)31 * 32 * num_sms) {   // one state per tile: 64 registers suffice -> 31 consumer warps
        if (vk == 2 && uni && n == 3) return launch_variant<BT, SPT, 3, 2, true, 31>(p, num_sms, st, grid_out);
        if (vk == 2 && n <= 4) return launch_variant<BT, SPT, 4, 2, false, 31>(p, num_sms, st, grid_out);   // cfg3: 0.72 -> 0.79
    }
    if (vk == 2) {
        if (uni && n == 3) return launch_variant<BT, SPT, 3, 2, true, kNwA>(p, num_sms, st, grid_out);   // honeycomb
        if (uni && n == 6) return launch_variant<BT, SPT, 6, 2, true, kNwB>(p, num_sms, st, grid_out);   // cubic
        if (n <= 4) return launch_variant<BT, SPT, 4, 2, false, kNwA>(p, num_sms, st, grid_out);         // e.g. vacancies
        return launch_variant<BT, SPT, 8, 2, false, 15>(p, num_sms, st, grid_out);
    }
    if (vk == 1) {
        if (BT == 1 && n <= 4) return launch_variant<BT, SPT, 4, 1, false, 23>(p, num_sms, st, grid_out);
        return launch_variant<BT, SPT, 8, 1, false, 15>(p, num_sms, st, grid_out);
    }
    if constexpr (BT == 8) {
        // Table small enough for shared memory (cfg4: 7,864 values = 126 KB): each block copies it once, the values are fetched
        // with LDS only when the gathers have returned (no registers held for them), which leaves room for all eight gathers
        // of a row in one round trip.  cfg4: 1955 -> 1885 us per launch.
        const size_t tab = (size_t)p.n_table * sizeof(double2);
        const size_t two_stages = 2 * (size_t)stage_geom(19 * 32 / (BT / SPT), n, true).stage_bytes;
        const bool tab_smem = uni && tab <= 150 * 1024 && tab + two_stages <= kSmemMax && knob("tab_smem", 1);
        if (tab_smem && n % 8 == 0) return launch_variant<BT, SPT, 8, 4, true, 15>(p, num_sms, st, grid_out);
        if (tab_smem && n % 4 == 0) return launch_variant<BT, SPT, 4, 4, true, 19>(p, num_sms, st, grid_out);
    }
    if (uni && n % 4 == 0) return launch_variant<BT, SPT, 4, 0, true, 15>(p, num_sms, st, grid_out);     // square + flux
    return launch_variant<BT, SPT, 4, 0, false, 15>(p, num_sms, st, grid_out);
}

}  // namespace ph
}  // namespace tbpm_detail

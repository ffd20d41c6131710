// term_pair.cuh -- TWO consecutive Chebyshev terms in one sweep of the vectors (temporal blocking through the L2).
//
//   phase 0:  T_k     = a0*H*T_{k-1} - T_{k-2}   (x = B, y = A: in place over T_{k-2})
//   phase 1:  T_{k+1} = a1*H*T_k     - T_{k-1}   (x = A, y = B: in place over T_{k-1})
//   either phase may also flush up to three terms into psi' and (phase 1 of the last pair) reduce <psi0|psi'>, <psi'|psi'>.
//
// Why: term_ph.cuh already moves the plain term's bytes at 80-92 % of the DRAM copy rate, so the only way to go faster is to
// move fewer bytes.  Two separate launches move 2 x (matrix + 3 vectors); here T_k, T_{k-1} and the matrix slices that phase 1
// needs were touched by phase 0 a few hundred tiles earlier and are still in the 126 MB L2: DRAM sees matrix + 4 vectors.
//
// How: the same block shape as term_ph.cuh (1 producer warp + NW consumer warps per SM, one block per SM, all co-resident --
// cooperative launch).  Tile t belongs to block t % G.  A block's work is a fixed SEQUENCE of items: step j issues phase 0 of
// its j-th tile, then phase 1 of its (j - lag)-th tile.  Phase 1 of tile t gathers T_k from, and overwrites T_{k-1} rows that
// are gathered by, the tiles within +-halo of t (halo = widest column offset in tiles, from the builder's lattice strides), so
// it must wait until phase 0 of all those tiles is finished: every block publishes the number of phase-0 tiles it has finished
// (st.release.gpu after a block-wide count of warps), and the producer warp of the waiting block polls the 148 counters
// (ld.acquire.gpu) before it releases the item's stage to its consumers.  lag >= ceil((halo + G) / G) + 1 makes every awaited
// item precede the waiting one in its owner's sequence, so the wait cannot deadlock.  Tiles whose dependency range wraps round
// the periodic boundary run phase 1 at the very end, after all of phase 0.
// Coherence: rows written in this launch are read back only through plain ld.global (no .nc), and the only earlier readers of
// the overwritten buffers inside the launch use L1::no_allocate loads, so no SM can hold a stale line of them.
#pragma once

#include <cooperative_groups.h>

#include "term_ph.cuh"

namespace tbpm_detail {
namespace pair {

using namespace ph;

constexpr int kPoll = 8;                 // counters polled per producer lane: grids of up to 256 blocks
constexpr int kRing = 2 * kMaxStages;    // per-item warp counters: warps of a block are never more than n_stage items apart

__device__ __forceinline__ int ld_acquire(const int *p)
{
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ int ld_relaxed(const int *p)
{
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(int *p, int v)
{
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

template <int SPT> struct CLoad;                            // coherent (L1-allocating, not .nc) loads of rows written in this launch
template <> struct CLoad<1> {
    static __device__ __forceinline__ void ld(CVec<1> &o, const double2 *p, bool on)
    {
        asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %3, 0;\nmov.f64 %0, 0d0000000000000000;\nmov.f64 %1, 0d0000000000000000;\n"
                     "@q ld.global.v2.f64 {%0, %1}, [%2];\n}"
                     : "=d"(o.v[0].x), "=d"(o.v[0].y)
                     : "l"(p), "r"((int)on)
                     : "memory");
    }
};
template <> struct CLoad<2> {
    static __device__ __forceinline__ void ld(CVec<2> &o, const double2 *p, bool on)
    {
        asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %5, 0;\nmov.f64 %0, 0d0000000000000000;\nmov.f64 %1, 0d0000000000000000;\n"
                     "mov.f64 %2, 0d0000000000000000;\nmov.f64 %3, 0d0000000000000000;\n"
                     "@q ld.global.v4.f64 {%0, %1, %2, %3}, [%4];\n}"
                     : "=d"(o.v[0].x), "=d"(o.v[0].y), "=d"(o.v[1].x), "=d"(o.v[1].y)
                     : "l"(p), "r"((int)on)
                     : "memory");
    }
};

// The item sequence of one block (identical in its producer and consumer warps).
struct ItemSeq {
    int64_t b, G, T, H, J, j, wi;
    int lag, sub, mode;
    __device__ __forceinline__ bool core(int64_t t) const { return t >= H && t <= T - 1 - H; }
    __device__ __forceinline__ void init(int64_t block, int64_t grid, int64_t n_tiles, int64_t halo, int lag_)
    {
        b = block; G = grid; T = n_tiles; H = halo; lag = lag_;
        J = b < T ? (T - b + G - 1) / G : 0;
        j = 0; sub = 0; mode = 0; wi = 0;
    }
    // next item: phase (0/1) and tile; false when the block is done
    __device__ __forceinline__ bool next(int &phase, int64_t &tile)
    {
        for (;;) {
            if (mode == 0) {
                if (j >= J + lag) { mode = 1; continue; }
                if (sub == 0) {
                    sub = 1;
                    if (j < J) { phase = 0; tile = b + j * G; return true; }
                } else {
                    sub = 0;
                    const int64_t i = j - lag;
                    ++j;
                    if (i >= 0 && i < J && core(b + i * G)) { phase = 1; tile = b + i * G; return true; }
                }
            } else {
                while (wi < J) {
                    const int64_t t = b + wi * G;
                    ++wi;
                    if (!core(t)) { phase = 1; tile = t; return true; }
                }
                return false;
            }
        }
    }
};

template <int BT, int SPT, int CH, int VK, bool UNI, int NW>
__global__ void __launch_bounds__((NW + 1) * 32, 1) k_term_pair(const PairParams q)
{
    constexpr int kConsumers = NW * 32;
    constexpr int LPR = BT / SPT;                           // lanes per row
    constexpr int R = kConsumers / LPR;                     // rows per tile
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t bars[2 * kMaxStages];  // [0, S): full, [kMaxStages, kMaxStages + S): empty
    __shared__ uint32_t lo_s[kMaxStages][2];                // first column / value-index element held by each stage
    __shared__ double red_s[NW][BT][3];
    __shared__ int ring[kRing];                             // warps that have finished the phase-0 item in this slot

    const TermParams &p = q.t;
    const int tid = threadIdx.x;
    const bool has_diag = p.diag != nullptr;
    const int S = p.n_stage;
    const int64_t n_tiles = (p.n_orb + R - 1) / R;
    const uint32_t bar0 = smem_u32(bars), smem0 = smem_u32(smem);
    const uint32_t n_uni = (uint32_t)p.max_row_off;

    if (tid == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(bar0 + 8 * s, 1); mbar_init(bar0 + 8 * (kMaxStages + s), kConsumers / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (tid < kRing) ring[tid] = 0;
    __syncthreads();

    ItemSeq seq;
    seq.init(blockIdx.x, gridDim.x, n_tiles, q.halo, q.lag);
    int phase = 0;
    int64_t tile = 0;

    if (tid >= kConsumers) {
        // ------------------------------------------------ producer warp ------------------------------------------------
        const int lane = tid & 31;
        const int64_t G = gridDim.x;
        int s = 0;
        uint32_t ph = 1;                                    // parity of the "empty" phase to wait for; first pass: free
        int seen[kPoll];                                    // last value read of the counters of blocks lane, lane + 32, ...
#pragma unroll
        for (int i = 0; i < kPoll; ++i) seen[i] = 0;
        while (seq.next(phase, tile)) {
            if (phase == 1) {                               // wait for phase 0 of every tile this item gathers from / overwrites
                const bool core = seq.core(tile);
                const int64_t upto = tile + q.halo;
                int req[kPoll];
#pragma unroll
                for (int i = 0; i < kPoll; ++i) {
                    const int64_t b2 = lane + 32 * i;
                    const int64_t jb = b2 < n_tiles && b2 < G ? (n_tiles - b2 + G - 1) / G : 0;
                    req[i] = (int)(core ? (upto >= b2 ? min(jb, (upto - b2) / G + 1) : 0) : jb);
                }
                unsigned spins = 0;
                // No acquire fence (it would invalidate the SM's L1 at every refresh): a counter value can only be seen after the
                // rows it announces reached L2 (release on the writer's side), no L1 can hold an older copy of those rows (see
                // the header), and the consumers' loads are issued after the mbarrier hand-off below.
                for (;;) {                                  // the counters only grow: the cached copies usually suffice
                    bool ok = true;
#pragma unroll
                    for (int i = 0; i < kPoll; ++i) ok = ok && seen[i] >= req[i];
                    if (__all_sync(0xffffffffu, ok)) break;
#pragma unroll
                    for (int i = 0; i < kPoll; ++i)
                        if (lane + 32 * i < G) seen[i] = ld_relaxed(q.progress + lane + 32 * i);
                    if (++spins > 8) __nanosleep(100);
                    if (spins > (1u << 22) || *(volatile int *)q.error) { *q.error = 1; break; }   // ~1 s: blocks not co-resident
                }
                __syncwarp();
            }
            if (lane == 0) {
                const int64_t r0 = tile * R;
                const int rows = (int)min((int64_t)R, p.n_orb - r0);
                uint32_t c_lo, c_hi;
                if (UNI) { c_lo = (uint32_t)r0 * n_uni; c_hi = c_lo + (uint32_t)rows * n_uni; }
                else { c_lo = __ldg(p.orp + r0); c_hi = __ldg(p.orp + r0 + rows); }
                const uint32_t full = bar0 + 8 * s;
                mbar_wait(bar0 + 8 * (kMaxStages + s), ph); // a fresh barrier reports the "previous" phase complete
                const uint32_t st = smem0 + (uint32_t)s * (uint32_t)p.stage_bytes;
                const uint32_t col_lo = c_lo & ~3u, idx_lo = c_lo & ~7u;
                const uint32_t nc = ((c_hi - col_lo) + 3u) & ~3u, ni = ((c_hi - idx_lo) + 7u) & ~7u;
                lo_s[s][0] = col_lo;
                lo_s[s][1] = idx_lo;
                uint32_t tx = 0;
                if (!UNI) {
                    const uint32_t orp_bytes = (uint32_t)(((rows + 1) * 4 + 15) & ~15);
                    bulk_g2s(st, p.orp + r0, orp_bytes, full);
                    tx += orp_bytes;
                }
                if (nc > 0) {
                    bulk_g2s(st + p.off_col, p.ocol + col_lo, nc * 4, full);
                    tx += nc * 4;
                    if (VK == 0) { bulk_g2s(st + p.off_idx, p.oidx + idx_lo, ni * 2, full); tx += ni * 2; }
                }
                if (has_diag) {
                    const uint32_t db = (uint32_t)((rows * 8 + 15) & ~15);
                    bulk_g2s(st + p.off_diag, p.diag + r0, db, full);
                    tx += db;
                }
                mbar_expect_tx(full, tx);                   // release: publishes lo_s[s] and, transitively, the acquired counters
            }
            __syncwarp();
            if (++s == S) { s = 0; ph ^= 1u; }
        }
        return;
    }

    // ---------------------------------------------------- consumer warps ----------------------------------------------------
    const int rl = tid / LPR;                               // row within the tile
    const int b0 = (tid % LPR) * SPT;                       // first state of this thread
    const uint32_t stage_bytes = (uint32_t)p.stage_bytes;
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

    // Rotated loop as in term_ph.cuh: an iteration consumes the chunk the previous one loaded, then loads the next.
    int s = 0, n_p0 = 0;                                    // n_p0: phase-0 items this warp has finished
    uint32_t ph = 0, so = 0;
    bool valid = false, more = false;
    int64_t e = 0;
    uint32_t n = 0, nmax = 0, c0 = 0, ca = 0, ia = 0;
    double d = 0.0;
    int cur = 0;                                            // phase of the item in flight
    const double2 *xb = nullptr;
    CVec<SPT> yold, xrow, aold, z, h;
    CVec<SPT> x[CH];
    double2 v[CH];
    uint32_t w[CH];

    auto load_row = [&]() {                                 // streamed operands + row header of (phase, tile)
        cur = phase;
        const PhaseParams &P = q.ph[cur];
        const int64_t row = tile * R + rl;
        valid = row < p.n_orb;
        e = row * BT + b0;
        xb = P.x + b0;
        const bool need_y = P.sub_y || P.n_acc == 3;
        const bool need_acc = P.n_acc > 0 && !P.acc_init;
        const bool need_xrow = P.n_acc >= 2 || has_diag;
        yold.stream_if(P.y + e, valid && need_y);           // own rows: T_{k-2} (phase 0) / T_{k-1} (phase 1), still unmodified
        aold.stream_if(p.acc + e, valid && need_acc);
        z.stream_if(p.psi0 + e, valid && P.reduce);
        CLoad<SPT>::ld(xrow, P.x + e, valid && need_xrow);  // phase 1: T_k of this very tile, written by this thread earlier
        mbar_wait(bar0 + 8 * s, ph);                        // phase 1: also "every tile within the halo has finished phase 0"
        if (UNI) {                                          // rows past the end of the last tile redo its first row, unstored
            const uint32_t rle = valid ? (uint32_t)rl : 0u;
            const uint32_t q0 = (uint32_t)(tile * R) * n_uni;
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
        uint32_t id[CH];
#pragma unroll
        for (int j = 0; j < CH; ++j) {
            const bool on = UNI || c0 + j < n;
            w[j] = lds_u32_if(ca + 4u * (c0 + j), on);
            id[j] = VK == 0 ? lds_u16_if(ia + 2u * (c0 + j), on) : 0u;
        }
        if (c0 + CH >= nmax) {                              // last chunk of every row of this warp: the stage is free again
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(bar0 + 8 * (kMaxStages + s));
            if (++s == S) { s = 0; ph ^= 1u; so = 0; } else so += stage_bytes;
        }
#pragma unroll
        for (int j = 0; j < CH; ++j) CLoad<SPT>::ld(x[j], xb + (int64_t)(w[j] & 0x7fffffffu) * BT, UNI || c0 + j < n);
        if (VK == 0) {
#pragma unroll
            for (int j = 0; j < CH; ++j) v[j] = table_value(ldg_value_if(p.vtab + (id[j] & 0x7fffu), UNI || c0 + j < n), id[j]);
        }
    };

    // Publication of a finished phase-0 item: every warp makes its own stores visible device-wide (a release store: MEMBAR,
    // no L1 invalidation), then counts itself in; the last warp of the block advances the block's counter.  It is delayed to
    // the epilogue of the warp's NEXT item, when those stores have long been acknowledged and the fence costs nothing.
    int pending = -1;
    auto publish = [&](int idx) {
        __syncwarp();
        if ((tid & 31) == 0) {
            st_release(q.progress + 2 * kMaxGrid + blockIdx.x * 32 + (tid >> 5), idx);   // per-warp scratch word: the release is the point
            const int slot = idx % kRing;
            if (atomicAdd(&ring[slot], 1) == NW - 1) {
                ring[slot] = 0;
                st_release(q.progress + blockIdx.x, idx + 1);
            }
        }
    };

    more = seq.next(phase, tile);
    if (more) {
        load_row();
        load_chunk();
    }
#pragma unroll 1
    while (more) {
        // ---- consume the chunk in flight, in issue order
        if (VK == 2) {
#pragma unroll
            for (int j = 0; j < CH; ++j) {
#pragma unroll
                for (int k = 0; k < SPT; ++k) { h.v[k].x += x[j].v[k].x; h.v[k].y += x[j].v[k].y; }
            }
        } else {
#pragma unroll
            for (int j = 0; j < CH; ++j) {
                if (VK == 1) v[j] = (w[j] >> 31) ? t1 : t0;
#pragma unroll
                for (int k = 0; k < SPT; ++k) cfma(h.v[k], v[j], x[j].v[k]);
            }
        }
        c0 += CH;
        if (c0 >= nmax) {
            // ---- epilogue of the row
            if (pending >= 0) { publish(pending); pending = -1; }   // the stores of that item left a whole item ago: cheap fence
            const PhaseParams &P = q.ph[cur];
            if (VK == 2) {
#pragma unroll
                for (int k = 0; k < SPT; ++k) { h.v[k].x *= t0.x; h.v[k].y *= t0.x; }
            }
            if (has_diag) {
#pragma unroll
                for (int k = 0; k < SPT; ++k) { h.v[k].x = fma(d, xrow.v[k].x, h.v[k].x); h.v[k].y = fma(d, xrow.v[k].y, h.v[k].y); }
            }
#pragma unroll
            for (int k = 0; k < SPT; ++k) { h.v[k].x *= P.a; h.v[k].y *= P.a; }
            if (P.sub_y) {
#pragma unroll
                for (int k = 0; k < SPT; ++k) { h.v[k].x -= yold.v[k].x; h.v[k].y -= yold.v[k].y; }
            }
            if (valid) {
                if (!P.reduce) h.st(P.y + e);               // T_k stays cacheable: phase 1 gathers it from L2
                if (P.n_acc > 0) {
#pragma unroll
                    for (int k = 0; k < SPT; ++k) {
                        cfma(aold.v[k], P.ca, h.v[k]);
                        if (P.n_acc >= 2) cfma(aold.v[k], P.cb, xrow.v[k]);
                        if (P.n_acc == 3) cfma(aold.v[k], P.cc, yold.v[k]);
                    }
                    if (P.reduce) {
#pragma unroll
                        for (int k = 0; k < SPT; ++k) {
                            s_re[k] = fma(z.v[k].x, aold.v[k].x, s_re[k]);      // conj(z) * psi'
                            s_re[k] = fma(z.v[k].y, aold.v[k].y, s_re[k]);
                            s_im[k] = fma(z.v[k].x, aold.v[k].y, s_im[k]);
                            s_im[k] = fma(-z.v[k].y, aold.v[k].x, s_im[k]);
                            s_nn[k] = fma(aold.v[k].x, aold.v[k].x, s_nn[k]);
                            s_nn[k] = fma(aold.v[k].y, aold.v[k].y, s_nn[k]);
                        }
                        aold.st(p.acc + e);
                    } else {
                        aold.st_stream(p.acc + e);
                    }
                }
            }
            if (cur == 0) {                                 // one more phase-0 tile of this warp is complete
                if (n_p0 + 1 >= seq.J) publish(n_p0);       // the block's last one: nothing later would carry the publication
                else pending = n_p0;
                ++n_p0;
            }
            more = seq.next(phase, tile);
            if (!more) break;
            load_row();
        }
        // ---- load: the next chunk (of this row, or the first of the next item's row)
        load_chunk();
    }

    if (q.ph[0].reduce || q.ph[1].reduce) {
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
            for (int w2 = 0; w2 < NW; ++w2) t += red_s[w2][bb][c];
            p.partial[((int64_t)blockIdx.x * BT + bb) * 3 + c] = t;
        }
    }
}

template <int BT, int SPT, int CH, int VK, bool UNI, int NW>
int launch_pair(PairParams q, int num_sms, cudaStream_t st, int *grid_out)
{
    constexpr int kConsumers = NW * 32, kThreads = kConsumers + 32;
    constexpr int R = kConsumers / (BT / SPT);
    TermParams &p = q.t;
    p.n_stage = std::min(kMaxStages, std::max(2, env_int("TBPM_STAGES", 4)));
    p.cap_entries = ((R * std::max(p.max_row_off, 1) + 8 + 7) / 8) * 8;
    size_t o = (size_t)(((R + 1) * 4 + 15) & ~15);
    p.off_col = (int)o;  o += (size_t)p.cap_entries * 4;
    p.off_idx = (int)o;  o += VK == 0 ? (size_t)p.cap_entries * 2 : 0;
    o = (o + 15) & ~size_t(15);
    p.off_diag = (int)o; o += (size_t)((R * 8 + 15) & ~15);
    p.stage_bytes = (int)((o + 127) & ~size_t(127));
    p.n_stage = (int)std::max<size_t>(2, std::min<size_t>(p.n_stage, (size_t)160 * 1024 / p.stage_bytes));
    const size_t dyn = (size_t)p.stage_bytes * p.n_stage;
    auto kern = k_term_pair<BT, SPT, CH, VK, UNI, NW>;
    static size_t configured = 0;
    if (dyn > configured) {
        const size_t want = std::max(dyn, (size_t)64 * 1024);
        TBPM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)want));
        configured = want;
    }
    const int64_t n_tiles = (p.n_orb + R - 1) / R;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>({n_tiles, (int64_t)num_sms, (int64_t)32 * kPoll}));
    // dependency geometry in tiles of THIS shape: +1 for the misalignment of a row offset with the tile grid
    q.halo = (q.halo + R - 1) / R + 1;                      // q.halo arrives in rows
    q.lag = (int)((q.halo + grid + grid - 1) / grid) + 1 + p.n_stage + env_int("TBPM_LAG_EXTRA", 0);   // + the producer's lead over its consumers
    TBPM_CUDA_TRY(cudaMemsetAsync(q.progress, 0, sizeof(int) * (size_t)grid, st));
    void *args[] = {&q};
    TBPM_CUDA_TRY(cudaLaunchCooperativeKernel((const void *)kern, dim3(grid), dim3(kThreads), args, dyn, st));   // all blocks resident
    count_launches(1);
    *grid_out = grid;
    return TBPM_OK;
}

// Rows per tile of the shape launch_pair_bt will pick (the caller sizes the L2 footprint with it).
template <int BT>
int launch_pair_bt(const PairParams &q, int num_sms, cudaStream_t st, int *grid_out)
{
    constexpr int SPT = 2;
    const TermParams &p = q.t;
    const int n = p.max_row_off;
    const bool uni = p.uniform;
    const int vk = p.single_real ? 2 : (p.packed ? 1 : 0);
    if (vk == 2) {
        if (uni && n == 3) return launch_pair<BT, SPT, 3, 2, true, 19>(q, num_sms, st, grid_out);
        if (uni && n == 6) return launch_pair<BT, SPT, 6, 2, true, 15>(q, num_sms, st, grid_out);
        if (n <= 4) return launch_pair<BT, SPT, 4, 2, false, 19>(q, num_sms, st, grid_out);
        return launch_pair<BT, SPT, 8, 2, false, 15>(q, num_sms, st, grid_out);
    }
    if (vk == 1) return launch_pair<BT, SPT, 8, 1, false, 15>(q, num_sms, st, grid_out);
    if (uni && n % 4 == 0) return launch_pair<BT, SPT, 4, 0, true, 15>(q, num_sms, st, grid_out);
    return launch_pair<BT, SPT, 4, 0, false, 15>(q, num_sms, st, grid_out);
}

}  // namespace pair
}  // namespace tbpm_detail

// term_rw.cu -- fused Chebyshev term on LATTICES: the vector rows a block needs arrive ONCE, by bulk copies (TMA), in a
// ROLLING WINDOW of shared memory, and the neighbours are read from it with LDS.  Tiles of 8 interleaved states.
//
//   T_k = a*H*T_{k-1} - T_{k-2}  (amxsy) + deferred psi' accumulation (axpy) + last-term
//   <psi0|psi'>, <psi'|psi'> (calc_corr_dos), exactly as term_ph.cuh; same TermParams, same results.
//
// Why (profiles/r2_ncu_cfg5.md, profiles/r1c_final.md): with 8 states a vector row is one 128-byte line, and the phased kernel
// asks the L1 for 9-10 lines per row (6-8 gathers, x[row], y, the store).  A line that misses L1 costs the SM 2.2 cycles of
// its L2 port, one that hits 0.84, and the registers that receive the gathers cap the loads in flight at ~130 KB per SM:
// 22-30 cycles per row where the HBM needs 15.8.  On a lattice almost all of those requests are redundant.  Let W be the
// largest lattice stride (a plane of the cubic lattice, a line of the square one) and let a block WALK along it: tile j+1
// of a run is tile j shifted by W rows.  Then the rows tile j gathers at +W are the own rows of tile j+1 and the -W
// neighbours of tile j+2, and the +-1 neighbours are the own rows shifted by one.  So:
//   ring   NR slots of R + 2 rows of x (R = 128 rows of the tile + one halo row on each side): per tile ONE new slot is
//          filled, by ONE 16 KB bulk copy, with the rows at +W; the slots of the previous two tiles serve 0 and -W;
//   stage  per tile: the column words / value indices / diagonal of its rows and its 128 rows of y (T_{k-2}), one bulk
//          copy each, n_stage tiles ahead;
//   consumers (16 warps, thread = row x 2 states) read every neighbour whose column IS row + delta_j from the ring with
//          two conflict-free LDS.128; entries that are not where the lattice puts them (periodic seams) and lattice offsets
//          that are neither near 0 nor near +-W (the +-line neighbours of the cubic lattice) are gathered with LDG.256 as
//          before.  psi' and psi0 (every third term / last term only) are streamed with LDG as in term_ph.cuh.
// Every row of x enters the SM once instead of three to nine times, no gather holds registers while it is in flight, and
// the DRAM sees 16 KB sequential bursts.  The offsets delta_j come from one sample row (build.cu, lat_delta); a matrix that
// does not follow them still gives the right answer through the LDG path, only slower.
#include <algorithm>

#include "term_ph.cuh"

namespace tbpm_detail {
namespace rw {

using namespace ph;

constexpr int kBT = 8, kNW = 16, kConsumers = kNW * 32, kThreads = kConsumers + 64, kR = kConsumers / 4;   // 128 rows per tile; two producer warps
constexpr int kHalo = 1;                                   // halo rows on each side of a ring slot
constexpr int kRowBytes = kBT * 16;
constexpr int kSlotBytes = (kR + 2 * kHalo) * kRowBytes;   // 16,640
constexpr int kMaxRing = 8, kMaxSlot = 8;
enum Src { SRC_PREV = 0, SRC_OWN = 1, SRC_NEXT = 2, SRC_GLOBAL = 3 };

struct Geom {
    int64_t W;                  // walk stride in rows (a multiple of kR that divides n_orb)
    int64_t d0;                 // tiles per lattice line, W / kR
    int64_t n_lines;            // n_orb / W
    int len;                    // tiles per run
    int n_ring, n_stage;
    int slot_delta[kMaxSlot];   // expected col - row of entry j
    int slot_src[kMaxSlot];     // where entry j is read: ring slot of tile j-1 / j / j+1, or global memory
    int slot_shift[kMaxSlot];   // row shift inside the ring slot, in [-kHalo, kHalo]
    int lat;                    // which Lat<> the (src, shift) pattern is, -1: none
    int far_na;                 // far neighbours loaded without L1 allocation
    int off_y, off_col, off_idx, off_diag, stage_bytes;
};

__device__ __forceinline__ void lds_c(double2 &v, uint32_t a)
{
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
}
__device__ __forceinline__ void lds_c_if(double2 &v, uint32_t a, bool on)     // zero when off
{
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %3, 0;\nmov.f64 %0, 0d0000000000000000;\nmov.f64 %1, 0d0000000000000000;\n"
                 "@q ld.shared.v2.f64 {%0, %1}, [%2];\n}"
                 : "=d"(v.x), "=d"(v.y)
                 : "r"(a), "r"((int)on));
}
__device__ __forceinline__ void ldg_pair(double2 &lo, double2 &hi, const double2 *p)
{
    asm volatile("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(lo.x), "=d"(lo.y), "=d"(hi.x), "=d"(hi.y) : "l"(p));
}
__device__ __forceinline__ void ldg_pair_na(double2 &lo, double2 &hi, const double2 *p)   // no L1 allocation
{
    asm volatile("ld.global.nc.L1::no_allocate.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(lo.x), "=d"(lo.y), "=d"(hi.x), "=d"(hi.y) : "l"(p));
}
__device__ __forceinline__ void ldg_pair_if(double2 &lo, double2 &hi, const double2 *p, bool on)   // keeps lo / hi when off
{
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %5, 0;\n@q ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];\n}"
                 : "+d"(lo.x), "+d"(lo.y), "+d"(hi.x), "+d"(hi.y)
                 : "l"(p), "r"((int)on));
}

// The lattices with an instantiation: where each entry of a row (in column order) is read, and its row shift in the slot.
//   LAT 0  simple cubic, 6 entries:            -W, far, -1, +1, far, +W          (far: the +-line neighbours, by LDG)
//   LAT 1  square + next-nearest, 8 entries:   -W-1, -W, -W+1, -1, +1, W-1, W, W+1
//   LAT 2  square / rectangular, 4 entries:    -W, -1, +1, +W
template <int LAT> struct Lat;
template <> struct Lat<0> {
    static constexpr int CH = 6;
    __host__ __device__ static constexpr int src(int j) { constexpr int t[6] = {SRC_PREV, SRC_GLOBAL, SRC_OWN, SRC_OWN, SRC_GLOBAL, SRC_NEXT}; return t[j]; }
    __host__ __device__ static constexpr int shift(int j) { constexpr int t[6] = {0, 0, -1, 1, 0, 0}; return t[j]; }
};
template <> struct Lat<1> {
    static constexpr int CH = 8;
    __host__ __device__ static constexpr int src(int j) { constexpr int t[8] = {SRC_PREV, SRC_PREV, SRC_PREV, SRC_OWN, SRC_OWN, SRC_NEXT, SRC_NEXT, SRC_NEXT}; return t[j]; }
    __host__ __device__ static constexpr int shift(int j) { constexpr int t[8] = {-1, 0, 1, -1, 1, -1, 0, 1}; return t[j]; }
};
template <> struct Lat<2> {
    static constexpr int CH = 4;
    __host__ __device__ static constexpr int src(int j) { constexpr int t[4] = {SRC_PREV, SRC_OWN, SRC_OWN, SRC_NEXT}; return t[j]; }
    __host__ __device__ static constexpr int shift(int j) { constexpr int t[4] = {0, -1, 1, 0}; return t[j]; }
};
template <int LAT> __host__ __device__ constexpr int n_far()
{
    int n = 0;
    for (int j = 0; j < Lat<LAT>::CH; ++j) n += Lat<LAT>::src(j) == SRC_GLOBAL;
    return n;
}

struct RingPos {                                            // slot and barrier parity of one ring load, advanced incrementally
    uint32_t i, ph;
    __device__ __forceinline__ void adv(uint32_t nr) { if (++i == nr) { i = 0; ph ^= 1u; } }
};

// LAT: the lattice (above); NACC / REDUCE / VK as in term_ph.cuh (VK 0: table index per entry, values from the L1-resident
// table; VK 2: one real value, neighbours summed and scaled once).
template <int LAT, int NACC, bool REDUCE, int VK>
__global__ void __launch_bounds__(kThreads, 1) k_term_rw(const TermParams p, const Geom g)
{
    using L = Lat<LAT>;
    constexpr int CH = L::CH;
    constexpr int NG = n_far<LAT>();
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t bars[2 * kMaxStages + 2 * kMaxRing];   // stage full | stage empty | ring full | ring empty
    __shared__ double red_s[REDUCE ? kNW : 1][REDUCE ? kBT : 1][3];

    const int tid = threadIdx.x;
    const bool sub_y = p.flags & F_SUB_Y;
    const bool need_y = sub_y || NACC == 3;
    const bool need_acc = NACC > 0 && !(p.flags & F_ACC_INIT);
    const bool has_diag = p.diag != nullptr;
    const bool need_xrow = NACC >= 2 || has_diag;
    const int S = g.n_stage;
    const uint32_t NR = (uint32_t)g.n_ring;
    const uint32_t bar0 = smem_u32(bars), smem0 = smem_u32(smem);
    const uint32_t b_sfull = bar0, b_sempty = bar0 + 8 * kMaxStages, b_rfull = bar0 + 16 * kMaxStages, b_rempty = b_rfull + 8 * kMaxRing;
    const uint32_t ring0 = smem0, stage0 = smem0 + NR * kSlotBytes;

    if (tid == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(b_sfull + 8 * s, 1); mbar_init(b_sempty + 8 * s, kNW); }
        for (uint32_t s = 0; s < NR; ++s) { mbar_init(b_rfull + 8 * s, 1); mbar_init(b_rempty + 8 * s, kNW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // Runs: run u covers the tiles at in-line position u % d0 of the lines [(u / d0) * len, (u / d0 + 1) * len); the runs are
    // dealt to the blocks round-robin, so the blocks sweep the lattice together (L2 locality of the remaining gathers).
    const int64_t n_runs = g.d0 * ((g.n_lines + g.len - 1) / g.len);

    if (tid >= kConsumers) {
        // ------------------------------- producers: one thread of each of the two producer warps -------------------------------
        // Warp kNW feeds the ring (rows of x, shared by three tiles each), warp kNW + 1 the stages (matrix slices and y of
        // one tile).  They wait on different "empty" barriers, so neither holds the other back: the ring runs n_ring - 3
        // tiles ahead of the consumers, the stages n_stage.
        if ((tid & 31) != 0) return;
        if (tid == kConsumers) {
            RingPos rp{0u, 1u};                             // next ring load: slot, parity of its "empty" phase (first pass: free)
            auto ring_load = [&](int64_t row0) {           // rows [row0 - halo, row0 + R + halo) of x, clipped to the vector
                mbar_wait(b_rempty + 8 * rp.i, rp.ph);
                const uint32_t full = b_rfull + 8 * rp.i;
                const int64_t lo = max(row0 - kHalo, (int64_t)0), hi = min(row0 + kR + kHalo, p.n_orb);
                uint32_t bytes = 0;
                if (row0 >= 0 && row0 < p.n_orb && hi > lo) {
                    bytes = (uint32_t)(hi - lo) * kRowBytes;
                    bulk_g2s(ring0 + rp.i * kSlotBytes + (uint32_t)(lo - (row0 - kHalo)) * kRowBytes, p.x + lo * kBT, bytes, full);
                }
                mbar_expect_tx(full, bytes);
                rp.adv(NR);
            };
            for (int64_t u = blockIdx.x; u < n_runs; u += gridDim.x) {
                const int64_t lb = u / g.d0, pos = u - lb * g.d0;
                const int64_t line0 = lb * g.len;
                const int len_u = (int)min((int64_t)g.len, g.n_lines - line0);
                const int64_t r_first = line0 * g.W + pos * kR;
                ring_load(r_first - g.W);
                ring_load(r_first);
                for (int j = 0; j < len_u; ++j) ring_load(r_first + (int64_t)(j + 1) * g.W);
            }
        } else {
            int s = 0;
            uint32_t sph = 1;
            for (int64_t u = blockIdx.x; u < n_runs; u += gridDim.x) {
                const int64_t lb = u / g.d0, pos = u - lb * g.d0;
                const int64_t line0 = lb * g.len;
                const int len_u = (int)min((int64_t)g.len, g.n_lines - line0);
                const int64_t r_first = line0 * g.W + pos * kR;
                for (int j = 0; j < len_u; ++j) {
                    const int64_t r0 = r_first + (int64_t)j * g.W;
                    mbar_wait(b_sempty + 8 * s, sph);
                    const uint32_t full = b_sfull + 8 * s;
                    const uint32_t st = stage0 + (uint32_t)s * (uint32_t)g.stage_bytes;
                    uint32_t tx = kR * CH * 4;
                    if (need_y) { bulk_g2s(st + g.off_y, p.y + r0 * kBT, kR * kRowBytes, full); tx += kR * kRowBytes; }
                    bulk_g2s(st + g.off_col, p.ocol + r0 * CH, kR * CH * 4, full);
                    if (VK == 0) { bulk_g2s(st + g.off_idx, p.oidx + r0 * CH, kR * CH * 2, full); tx += kR * CH * 2; }
                    if (has_diag) { bulk_g2s(st + g.off_diag, p.diag + r0, kR * 8, full); tx += kR * 8; }
                    mbar_expect_tx(full, tx);
                    if (++s == S) { s = 0; sph ^= 1u; }
                }
            }
        }
        return;
    }

    // ---------------------------------------------------- consumer warps ----------------------------------------------------
    const int rl = tid >> 2, q = tid & 3, par = rl & 1;     // row of the tile, lane of the row, row parity
    // Odd rows read their two 16-byte halves in the opposite order: a quarter-warp (2 rows x 4 lanes) then touches all 32 banks.
    // Slot "a" of a thread is state 2q + par, slot "b" is state 2q + 1 - par.
    const uint32_t oa = (uint32_t)(2 * q + par) * 16u, ob = (uint32_t)(2 * q + 1 - par) * 16u;
    const uint32_t row_off = (uint32_t)(rl + kHalo) * kRowBytes;
    const uint32_t lane_off = (uint32_t)rl * kRowBytes;
    double2 t0 = make_double2(0.0, 0.0);
    if (VK == 2) t0 = __ldg(p.vtab);
    double sa_re = 0.0, sa_im = 0.0, sa_nn = 0.0, sb_re = 0.0, sb_im = 0.0, sb_nn = 0.0;
    int d_far[NG > 0 ? NG : 1];                             // lattice offsets of the far entries
    {
        int k = 0;
#pragma unroll
        for (int jj = 0; jj < CH; ++jj)
            if (L::src(jj) == SRC_GLOBAL) d_far[k++] = g.slot_delta[jj];
    }
    const int64_t last_row = p.n_orb - 1;

    RingPos r0p{0u, 0u}, r1p{1u % NR, 0u}, r2p{2u % NR, 0u};   // the ring loads holding the -W rows / own rows / +W rows of the tile
    if (NR <= 2) { r2p.i = 0; r2p.ph = 1; }                    // (NR >= 4 always; keeps the compiler honest)
    int s = 0;
    uint32_t sph = 0, st = stage0;
    // far neighbours of the NEXT tile are requested one tile ahead, at the columns the lattice predicts (natural state order)
    double2 fa[NG > 0 ? NG : 1], fb[NG > 0 ? NG : 1];
    auto far_request = [&](int64_t row) {
#pragma unroll
        for (int k = 0; k < NG; ++k) {
            int64_t c = row + d_far[k];
            c = c < 0 ? 0 : (c > last_row ? last_row : c);  // a clamped prediction is never confirmed (see the check below)
            if (g.far_na) ldg_pair_na(fa[k], fb[k], p.x + c * kBT + 2 * q); else ldg_pair(fa[k], fb[k], p.x + c * kBT + 2 * q);
        }
    };
    if (NG > 0 && (int64_t)blockIdx.x < n_runs) {
        const int64_t lb = blockIdx.x / g.d0, pos = blockIdx.x - lb * g.d0;
        far_request(lb * g.len * g.W + pos * kR + rl);
    }
#pragma unroll 1
    for (int64_t u = blockIdx.x; u < n_runs; u += gridDim.x) {
        const int64_t lb = u / g.d0, pos = u - lb * g.d0;
        const int64_t line0 = lb * g.len;
        const int len_u = (int)min((int64_t)g.len, g.n_lines - line0);
        int64_t row = line0 * g.W + pos * kR + rl;
        // first row of the next run of this block (for the far request of this run's last tile)
        int64_t next_run_row = -1;
        if (NG > 0 && u + gridDim.x < n_runs) {
            const int64_t u2 = u + gridDim.x, lb2 = u2 / g.d0, pos2 = u2 - lb2 * g.d0;
            next_run_row = lb2 * g.len * g.W + pos2 * kR + rl;
        }
#pragma unroll 1
        for (int j = 0; j < len_u; ++j, row += g.W) {
            const int64_t e = row * kBT + 2 * q;
            // ---- streamed operands that need no index and are not staged (HBM latency: issue first)
            CVec<2> aold, z;
            if (NACC > 0) aold.stream_if(p.acc + e, need_acc);
            if (REDUCE) z.stream_if(p.psi0 + e, true);
            // ---- wait: the ring slots of this tile (the first tile of a run waits for all three), then the stage
            if (j == 0) {
                mbar_wait(b_rfull + 8 * r0p.i, r0p.ph);
                mbar_wait(b_rfull + 8 * r1p.i, r1p.ph);
            }
            mbar_wait(b_rfull + 8 * r2p.i, r2p.ph);
            mbar_wait(b_sfull + 8 * s, sph);
            // ---- column words (and value indices) of the row; is every entry where the lattice puts it?
            uint32_t w[CH], id[CH];
            const uint32_t ca = st + g.off_col + (uint32_t)rl * (CH * 4u);
            const uint32_t ia = st + g.off_idx + (uint32_t)rl * (CH * 2u);
#pragma unroll
            for (int jj = 0; jj < CH; jj += 2) {
                lds_v2_u32(ca + 4u * jj, w[jj], w[jj + 1]);
                if (VK == 0) { const uint32_t t = lds_u32(ia + 2u * jj); id[jj] = t & 0xffffu; id[jj + 1] = t >> 16; }
                else id[jj] = id[jj + 1] = 0u;
            }
            const int row32 = (int)row;
            bool ok = true;
#pragma unroll
            for (int jj = 0; jj < CH; ++jj) ok = ok && ((int)(w[jj] & 0x7fffffffu) == row32 + g.slot_delta[jj]);
            const bool fast = __all_sync(0xffffffffu, ok);
            const uint32_t bp = ring0 + r0p.i * kSlotBytes + row_off, bo = ring0 + r1p.i * kSlotBytes + row_off,
                           bn = ring0 + r2p.i * kSlotBytes + row_off;
            double2 ha = make_double2(0.0, 0.0), hb = ha;   // slots a / b
            double2 ga = ha, gb = ha;                       // far neighbours, natural state order (2q, 2q + 1)
            if (fast) {
#pragma unroll
                for (int c0 = 0; c0 < CH; c0 += 4) {
                    double2 xa[4], xb[4], v[4];
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int jj = c0 + i < CH ? c0 + i : 0;
                        if (c0 + i >= CH || L::src(jj) == SRC_GLOBAL) continue;
                        const uint32_t a = (L::src(jj) == SRC_PREV ? bp : (L::src(jj) == SRC_OWN ? bo : bn)) + (uint32_t)(L::shift(jj) * kRowBytes);
                        lds_c(xa[i], a + oa);
                        lds_c(xb[i], a + ob);
                        if (VK == 0) v[i] = table_value(__ldg(p.vtab + (id[jj] & 0x7fffu)), id[jj]);
                    }
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int jj = c0 + i < CH ? c0 + i : 0;
                        if (c0 + i >= CH || L::src(jj) == SRC_GLOBAL) continue;
                        if (VK == 2) { ha.x += xa[i].x; ha.y += xa[i].y; hb.x += xb[i].x; hb.y += xb[i].y; }
                        else { cfma(ha, v[i], xa[i]); cfma(hb, v[i], xb[i]); }
                    }
                }
                {
                    int k = 0;
#pragma unroll
                    for (int jj = 0; jj < CH; ++jj)
                        if (L::src(jj) == SRC_GLOBAL) {
                            if (VK == 2) { ga.x += fa[k].x; ga.y += fa[k].y; gb.x += fb[k].x; gb.y += fb[k].y; }
                            else {
                                const double2 vv = table_value(__ldg(p.vtab + (id[jj] & 0x7fffu)), id[jj]);
                                cfma(ga, vv, fa[k]); cfma(gb, vv, fb[k]);
                            }
                            ++k;
                        }
                }
            } else {
                // a row of this warp sits on a periodic seam (or the matrix does not follow the lattice): entry by entry
                int k = 0;
#pragma unroll
                for (int jj = 0; jj < CH; ++jj) {
                    const int64_t col = (int64_t)(w[jj] & 0x7fffffffu);
                    const bool hit = (int)col == row32 + g.slot_delta[jj];
                    double2 v1 = t0;
                    if (VK == 0) v1 = table_value(__ldg(p.vtab + (id[jj] & 0x7fffu)), id[jj]);
                    if (L::src(jj) == SRC_GLOBAL) {
                        double2 x0 = fa[k], x1 = fb[k];
                        if (!hit) ldg_pair(x0, x1, p.x + col * kBT + 2 * q);
                        if (VK == 2) { ga.x += x0.x; ga.y += x0.y; gb.x += x1.x; gb.y += x1.y; }
                        else { cfma(ga, v1, x0); cfma(gb, v1, x1); }
                        ++k;
                    } else if (hit) {
                        const uint32_t a = (L::src(jj) == SRC_PREV ? bp : (L::src(jj) == SRC_OWN ? bo : bn)) + (uint32_t)(L::shift(jj) * kRowBytes);
                        double2 x0, x1;
                        lds_c(x0, a + oa);
                        lds_c(x1, a + ob);
                        if (VK == 2) { ha.x += x0.x; ha.y += x0.y; hb.x += x1.x; hb.y += x1.y; }
                        else { cfma(ha, v1, x0); cfma(hb, v1, x1); }
                    } else {
                        double2 x0, x1;
                        ldg_pair(x0, x1, p.x + col * kBT + 2 * q);
                        if (VK == 2) { ga.x += x0.x; ga.y += x0.y; gb.x += x1.x; gb.y += x1.y; }
                        else { cfma(ga, v1, x0); cfma(gb, v1, x1); }
                    }
                }
            }
            double2 ya = make_double2(0.0, 0.0), yb = ya, xra = ya, xrb = ya;
            if (need_y) { lds_c(ya, st + g.off_y + lane_off + oa); lds_c(yb, st + g.off_y + lane_off + ob); }
            if (need_xrow) { lds_c(xra, bo + oa); lds_c(xrb, bo + ob); }
            double d = has_diag ? lds_f64(st + g.off_diag + (uint32_t)rl * 8u) : 0.0;
            // the far sums are in natural state order: fold them into slots a / b
            ha.x += par ? gb.x : ga.x; ha.y += par ? gb.y : ga.y;
            hb.x += par ? ga.x : gb.x; hb.y += par ? ga.y : gb.y;
            // ---- request the far neighbours of the next tile (of this run, or of the block's next run)
            if (NG > 0) {
                const int64_t nrow = j + 1 < len_u ? row + g.W : next_run_row;
                if (nrow >= 0) far_request(nrow);
            }
            if (VK == 2) { ha.x *= t0.x; ha.y *= t0.x; hb.x *= t0.x; hb.y *= t0.x; }
            // Every shared-memory read of this tile must have RETURNED before the stage and the oldest ring slot are handed back to
            // the producers.  A load has returned once an instruction has read its destination register, so the barrier addresses
            // below are made to depend on all of them (`rel` is 0: p.zero is 0, but only at run time).
            const uint32_t rel = (uint32_t)(__double2hiint(ya.x) ^ __double2hiint(yb.x) ^ __double2hiint(xra.x) ^ __double2hiint(xrb.x) ^
                                            __double2hiint(d) ^ __double2hiint(ha.x) ^ __double2hiint(hb.x)) & (uint32_t)p.zero;
            __syncwarp();
            if ((tid & 31) == 0) {
                mbar_arrive(b_sempty + 8 * s + rel);
                mbar_arrive(b_rempty + 8 * r0p.i + rel);
                if (j == len_u - 1) { mbar_arrive(b_rempty + 8 * r1p.i + rel); mbar_arrive(b_rempty + 8 * r2p.i + rel); }
            }
            if (++s == S) { s = 0; sph ^= 1u; st = stage0; } else st += (uint32_t)g.stage_bytes;
            r0p.adv(NR); r1p.adv(NR); r2p.adv(NR);

            if (has_diag) { ha.x = fma(d, xra.x, ha.x); ha.y = fma(d, xra.y, ha.y); hb.x = fma(d, xrb.x, hb.x); hb.y = fma(d, xrb.y, hb.y); }
            ha.x *= p.a; ha.y *= p.a; hb.x *= p.a; hb.y *= p.a;
            if (sub_y) { ha.x -= ya.x; ha.y -= ya.y; hb.x -= yb.x; hb.y -= yb.y; }
            CVec<2> out;
            if (!REDUCE) {
                out.v[0] = par ? hb : ha; out.v[1] = par ? ha : hb;
                out.st_stream(p.y + e);                     // T_k: its readers come a whole sweep later
            }
            if (NACC > 0) {
                double2 aa = par ? aold.v[1] : aold.v[0], ab = par ? aold.v[0] : aold.v[1];
                cfma(aa, p.ca, ha); cfma(ab, p.ca, hb);
                if (NACC >= 2) { cfma(aa, p.cb, xra); cfma(ab, p.cb, xrb); }
                if (NACC == 3) { cfma(aa, p.cc, ya); cfma(ab, p.cc, yb); }
                out.v[0] = par ? ab : aa; out.v[1] = par ? aa : ab;
                if (REDUCE) {
                    const double2 za = par ? z.v[1] : z.v[0], zb = par ? z.v[0] : z.v[1];
                    sa_re = fma(za.x, aa.x, sa_re); sa_re = fma(za.y, aa.y, sa_re);
                    sa_im = fma(za.x, aa.y, sa_im); sa_im = fma(-za.y, aa.x, sa_im);
                    sa_nn = fma(aa.x, aa.x, sa_nn); sa_nn = fma(aa.y, aa.y, sa_nn);
                    sb_re = fma(zb.x, ab.x, sb_re); sb_re = fma(zb.y, ab.y, sb_re);
                    sb_im = fma(zb.x, ab.y, sb_im); sb_im = fma(-zb.y, ab.x, sb_im);
                    sb_nn = fma(ab.x, ab.x, sb_nn); sb_nn = fma(ab.y, ab.y, sb_nn);
                    out.st(p.acc + e);                      // psi': T_0 of the next step
                } else {
                    out.st_stream(p.acc + e);
                }
            }
        }
        r0p.adv(NR); r0p.adv(NR); r1p.adv(NR); r1p.adv(NR); r2p.adv(NR); r2p.adv(NR);   // a run of len tiles consumes len + 2 ring loads
    }

    if (REDUCE) {
        // slot a is state 2q + par, slot b is state 2q + 1 - par: put the sums in state order before the warp reduction
        double s_re[2] = {par ? sb_re : sa_re, par ? sa_re : sb_re};
        double s_im[2] = {par ? sb_im : sa_im, par ? sa_im : sb_im};
        double s_nn[2] = {par ? sb_nn : sa_nn, par ? sa_nn : sb_nn};
#pragma unroll
        for (int k = 0; k < 2; ++k) {
#pragma unroll
            for (int o = 16; o >= 4; o >>= 1) {
                s_re[k] += __shfl_xor_sync(0xffffffffu, s_re[k], o);
                s_im[k] += __shfl_xor_sync(0xffffffffu, s_im[k], o);
                s_nn[k] += __shfl_xor_sync(0xffffffffu, s_nn[k], o);
            }
        }
        const int lane = tid & 31, warp = tid >> 5;
        if (lane < 4) {
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                red_s[warp][lane * 2 + k][0] = s_re[k];
                red_s[warp][lane * 2 + k][1] = s_im[k];
                red_s[warp][lane * 2 + k][2] = s_nn[k];
            }
        }
        asm volatile("bar.sync 1, %0;" ::"n"(kConsumers) : "memory");   // consumers only (the producer warp has left)
        if (tid < kBT * 3) {
            const int bb = tid / 3, c = tid % 3;
            double t = 0.0;
#pragma unroll
            for (int w2 = 0; w2 < kNW; ++w2) t += red_s[w2][bb][c];
            p.partial[((int64_t)blockIdx.x * kBT + bb) * 3 + c] = t;
        }
    }
}

// Walk stride, entry sources and stage layout from the sample row's offsets.  false when the offsets do not describe a
// lattice this kernel is meant for.
bool make_geom(const TermParams &p, Geom &g)
{
    const int n = p.max_row_off;
    if (!p.uniform || p.n_table <= 0 || p.n_lat_off != n || (n != 4 && n != 6 && n != 8)) return false;
    if (p.n_orb <= 0 || p.n_orb >= ((int64_t)1 << 31)) return false;
    // W: the largest offset that is a whole number of tiles and divides the vector
    int64_t W = 0;
    for (int j = 0; j < n; ++j) {
        const int64_t d = p.lat_delta[j] < 0 ? -p.lat_delta[j] : p.lat_delta[j];
        if (d > kHalo && d % kR == 0 && p.n_orb % d == 0 && p.n_orb / d >= 4 && d > W) W = d;
    }
    if (W == 0) return false;
    g.W = W; g.d0 = W / kR; g.n_lines = p.n_orb / W;
    g.len = (int)std::min<int64_t>(std::max(1, knob("rw_len", 64)), g.n_lines);
    int n_global = 0;
    g.lat = -1;
    for (int j = 0; j < n; ++j) {
        const int64_t d = p.lat_delta[j];
        if (d == 0 || d > ((int64_t)1 << 30) || d < -((int64_t)1 << 30)) return false;
        g.slot_delta[j] = (int)d;
        if (d >= -kHalo && d <= kHalo) { g.slot_src[j] = SRC_OWN; g.slot_shift[j] = (int)d; }
        else if (d - W >= -kHalo && d - W <= kHalo) { g.slot_src[j] = SRC_NEXT; g.slot_shift[j] = (int)(d - W); }
        else if (d + W >= -kHalo && d + W <= kHalo) { g.slot_src[j] = SRC_PREV; g.slot_shift[j] = (int)(d + W); }
        else { g.slot_src[j] = SRC_GLOBAL; g.slot_shift[j] = 0; ++n_global; }
    }
    if (n_global > 2) return false;                        // then the phased kernel is the better shape
    auto same = [&](int (*src)(int), int (*shift)(int), int ch) {
        if (ch != n) return false;
        for (int j = 0; j < n; ++j)
            if (src(j) != g.slot_src[j] || (src(j) != SRC_GLOBAL && shift(j) != g.slot_shift[j])) return false;
        return true;
    };
    if (same(Lat<0>::src, Lat<0>::shift, Lat<0>::CH)) g.lat = 0;
    else if (same(Lat<1>::src, Lat<1>::shift, Lat<1>::CH)) g.lat = 1;
    else if (same(Lat<2>::src, Lat<2>::shift, Lat<2>::CH)) g.lat = 2;
    else return false;
    const bool with_idx = !(p.single_real || p.packed);
    size_t o = 0;
    g.off_y = (int)o;   o += (size_t)kR * kRowBytes;
    g.off_col = (int)o; o += (size_t)kR * n * 4;
    g.off_idx = (int)o; o += with_idx ? (size_t)kR * n * 2 : 0;
    g.off_diag = (int)o; o += (size_t)kR * 8;
    g.stage_bytes = (int)((o + 127) & ~size_t(127));
    g.far_na = knob("rw_far_na", 1);
    g.n_ring = std::min(kMaxRing, std::max(4, knob("rw_ring", 5)));
    g.n_stage = std::min(kMaxStages, std::max(2, knob("rw_stages", 4)));
    while ((size_t)g.n_ring * kSlotBytes + (size_t)g.n_stage * g.stage_bytes > kSmemMax - 4096) {
        if (g.n_stage > 2) --g.n_stage;
        else if (g.n_ring > 4) --g.n_ring;
        else return false;
    }
    return true;
}

template <int LAT, int NACC, bool REDUCE, int VK>
int launch_one(const TermParams &p, const Geom &g, int num_sms, cudaStream_t st, int *grid_out)
{
    const size_t dyn = (size_t)g.n_ring * kSlotBytes + (size_t)g.n_stage * g.stage_bytes;
    auto kern = k_term_rw<LAT, NACC, REDUCE, VK>;
    static size_t configured[kMaxDevices] = {0};
    if (p.device < 0 || p.device >= kMaxDevices) return TBPM_EINVAL;
    if (dyn > configured[p.device]) {
        TBPM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kSmemMax - 4096)));
        configured[p.device] = kSmemMax - 4096;
    }
    const int64_t n_runs = g.d0 * ((g.n_lines + g.len - 1) / g.len);
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>({n_runs, (int64_t)num_sms, (int64_t)kMaxGrid}));
    kern<<<grid, kThreads, dyn, st>>>(p, g);
    count_launches(1);
    *grid_out = grid;
    return TBPM_OK;
}

template <int LAT, int VK>
int launch_variant(const TermParams &p, const Geom &g, int num_sms, cudaStream_t st, int *grid_out)
{
    const bool red = p.flags & F_REDUCE;
    if (!red && p.n_acc == 0) return launch_one<LAT, 0, false, VK>(p, g, num_sms, st, grid_out);
    if (!red && p.n_acc == 3) return launch_one<LAT, 3, false, VK>(p, g, num_sms, st, grid_out);
    if (red && p.n_acc == 1) return launch_one<LAT, 1, true, VK>(p, g, num_sms, st, grid_out);
    if (red && p.n_acc == 2) return launch_one<LAT, 2, true, VK>(p, g, num_sms, st, grid_out);
    if (red && p.n_acc == 3) return launch_one<LAT, 3, true, VK>(p, g, num_sms, st, grid_out);
    return TBPM_EINVAL;
}

}  // namespace rw

bool term_rw_supported(int bt, const TermParams &p)
{
    if (bt != rw::kBT || (p.flags & F_SKIP_H) || !knob("rw", 1)) return false;
    const bool red = p.flags & F_REDUCE, wy = p.flags & F_WRITE_Y;
    if (red == wy) return false;
    if (!red && !(p.n_acc == 0 || p.n_acc == 3)) return false;
    if (red && (p.n_acc < 1 || p.n_acc > 3)) return false;
    if (p.packed && !p.single_real) return false;          // one complex value with conjugate bits: the phased kernel has that shape
    rw::Geom g;
    return rw::make_geom(p, g);
}

int launch_term_rw(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    rw::Geom g;
    if (!rw::make_geom(p, g)) return TBPM_EINVAL;
    switch (g.lat) {
    case 0: return p.single_real ? rw::launch_variant<0, 2>(p, g, num_sms, st, grid_out) : rw::launch_variant<0, 0>(p, g, num_sms, st, grid_out);
    case 1: return p.single_real ? rw::launch_variant<1, 2>(p, g, num_sms, st, grid_out) : rw::launch_variant<1, 0>(p, g, num_sms, st, grid_out);
    case 2: return p.single_real ? rw::launch_variant<2, 2>(p, g, num_sms, st, grid_out) : rw::launch_variant<2, 0>(p, g, num_sms, st, grid_out);
    }
    return TBPM_EINVAL;
}

}  // namespace tbpm_detail

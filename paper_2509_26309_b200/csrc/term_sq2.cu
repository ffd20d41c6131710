// term_sq2.cu -- TWO Chebyshev terms per sweep on the periodic square lattice with next-nearest neighbours and in-line hoppings
// (BASELINE.json:configs[3]; the lattice of term_sq.cu, tiles of 8 interleaved states; a real diagonal rides in the y stage).
//
//   T_k     = a1*H*T_{k-1} - T_{k-2}      (amxsy)
//   T_{k+1} = a2*H*T_k     - T_{k-1}
//   psi'   += ca*T_{k+1} + cb*T_k + cc*T_{k-1} + cd*T_{k-2}   (the axpy of PAPER.md:440 for up to FOUR terms at once), and on the last
//   pair of a time step <psi0|psi'>, <psi'|psi'> (calc_corr_dos).
//
// Why: term_sq.cu runs at the DRAM bandwidth (profiles/r2_ncu_cfg4.md), so the only way on is to move fewer bytes.  One term reads
// T_{k-1} and T_{k-2} and writes T_k: 3 vectors.  Here a block walks DOWN the lattice at a fixed in-line position, as in term_sq.cu,
// and keeps the last three lines of T_k it has just computed in a second shared-memory ring: T_{k+1} of line L - 1 follows as soon
// as T_k of line L exists.  A pair of terms then reads 2 vectors and writes 2 (4 instead of 6), and psi' is touched once per FOUR
// terms instead of three: 52 instead of 74 vector transfers per time step of 20 terms.
//   halo     T_{k+1} on rows [x0, x0 + 128) needs T_k on [x0 - 1, x0 + 129), from T_{k-1} on [x0 - 2, x0 + 130) -- ring slots of 132
//            rows -- and T_{k-2} on 130 rows; the two rows outside the tile are computed by a light "halo warp" (lane = row, state,
//            half of the directions).  Along the walk T_k is computed on one extra line above and below the run of 64 lines (+3 %).
//   buffers  T_{k-2} is now read with a halo, so T_k cannot overwrite it in place: both results go to buffers of their own
//            (TermParams::out1 / out2), which the next pair reads while it writes the two this pair read.
//   sync     8 main consumer warps (64 row pairs x 4 lanes; thread = 2 states of 2 adjacent rows, the values of those two rows in
//            registers for a whole run, serving both stages) + the halo warp.  Per line: stage 1 -> named barrier (the line of T_k
//            is in ring B) -> stage 2.  Ring B slot (it % 4) is rewritten two barriers after its last reader passed one: no
//            further hand-shake.  (A ninth FULL warp for a 65th row pair cost what the pairing won: 9 warps over 4 schedulers.)
//   less shared memory is faster here: it is L1 taken from the streamed stores (4 ring slots + 3 stages, not 5 + 4).
#include <algorithm>

#include "term_ph.cuh"

namespace tbpm_detail {
namespace sq2 {

using namespace ph;

constexpr int kBT = 8, kMainW = 8, kMain = kMainW * 32;    // main consumers: 64 row pairs x 4 lanes
constexpr int kNW = kMainW + 1, kConsumers = kNW * 32;     // + the halo warp
constexpr int kThreads = kConsumers + 64;                  // + two producer warps
constexpr int kR = 128;                                    // rows of a tile that this block OWNS (stores)
constexpr int kRowBytes = kBT * 16;
constexpr int kSlotRows = kR + 4;                          // tile rows -2 .. 129
constexpr int kSlotBytes = kSlotRows * kRowBytes;          // 16,896
constexpr int kYRows = kR + 2;                             // tile rows -1 .. 128
constexpr int kYBytes = kYRows * kRowBytes;                // 16,640
constexpr int kDiagRows = kR + 4;                          // diagonal of tile rows -2 .. 129 (16-byte aligned bulk copies), behind the y rows
constexpr int kDiagBytes = 1152;                           // 132 x 8 = 1,056, padded to a multiple of 128
constexpr int kMaxRing = 8;
constexpr int kNB = 4;                                     // slots of the T_k ring
constexpr int kCH = 8;

struct Geom {
    int64_t W, d0, n_lines;
    int len, n_ring, n_stage, stage_bytes;
};

struct RingPos {
    uint32_t i, ph;
    __device__ __forceinline__ void adv(uint32_t nr) { if (++i == nr) { i = 0; ph ^= 1u; } }
};

__device__ __forceinline__ void lds_c(double2 &v, uint32_t a)
{
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
}
// producer-side wait: poll with a pause, so that the spinning thread does not take issue slots from the consumer warps of its
// scheduler (a fifth of all issued instructions were these polls)
__device__ __forceinline__ void mbar_wait_idle(uint32_t bar, uint32_t parity)
{
    uint32_t done;
    for (;;) {
        asm volatile("{\n.reg .pred q;\nmbarrier.try_wait.parity.shared::cta.b64 q, [%1], %2;\nselp.u32 %0, 1, 0, q;\n}"
                     : "=r"(done)
                     : "r"(bar), "r"(parity)
                     : "memory");
        if (done) break;
        __nanosleep(400);
    }
}
__device__ __forceinline__ void sts_c(uint32_t a, double2 v)
{
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(a), "d"(v.x), "d"(v.y) : "memory");
}

struct Row2 { double2 a, b; };                             // the thread's two states of one row (slot a / slot b, see `par`)
struct Out4 { double2 Aa, Ab, Ba, Bb; };                   // rows A and B, slots a and b

// H * v on the thread's two rows from three consecutive lines held in 132-row slots (bp / bo / bn: address of slot row 2p of the
// line above / the own line / the line below); xA, xB return the own rows of the middle line.
// RX: the two in-line hops (directions 3, 4) are REAL (Landau gauge along the line, certified by the builder): 2 FMAs instead of 4;
// the result is the same bit for bit, the dropped FMAs would add 0 * x.
template <bool RX>
__device__ __forceinline__ void apply_h(uint32_t bp, uint32_t bo, uint32_t bn, uint32_t oa, uint32_t ob, const double2 (&vA)[kCH],
                                        const double2 (&vB)[kCH], Out4 &h, Row2 &xA, Row2 &xB)
{
    h.Aa = h.Ab = h.Ba = h.Bb = make_double2(0.0, 0.0);
    Row2 r[4];
    auto load4 = [&](uint32_t base) {                      // rows A - 1, A, B, B + 1 of one line
#pragma unroll
        for (int i = 0; i < 4; ++i) { lds_c(r[i].a, base + (uint32_t)i * kRowBytes + oa); lds_c(r[i].b, base + (uint32_t)i * kRowBytes + ob); }
    };
    load4(bp);                                             // line above: directions 0, 1, 2 = in-line offsets -1, 0, +1
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        cfma(h.Aa, vA[k], r[k].a); cfma(h.Ab, vA[k], r[k].b);
        cfma(h.Ba, vB[k], r[k + 1].a); cfma(h.Bb, vB[k], r[k + 1].b);
    }
    load4(bo);                                             // own line: directions 3, 4 = -1, +1; r[1], r[2] are the own rows
    auto hop = [](double2 &acc, double2 v, double2 x) {
        if (RX) { acc.x = fma(v.x, x.x, acc.x); acc.y = fma(v.x, x.y, acc.y); } else cfma(acc, v, x);
    };
    hop(h.Aa, vA[3], r[0].a); hop(h.Ab, vA[3], r[0].b);
    hop(h.Ba, vB[3], r[1].a); hop(h.Bb, vB[3], r[1].b);
    hop(h.Aa, vA[4], r[2].a); hop(h.Ab, vA[4], r[2].b);
    hop(h.Ba, vB[4], r[3].a); hop(h.Bb, vB[4], r[3].b);
    xA = r[1]; xB = r[2];
    load4(bn);                                             // line below: directions 5, 6, 7
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        cfma(h.Aa, vA[5 + k], r[k].a); cfma(h.Ab, vA[5 + k], r[k].b);
        cfma(h.Ba, vB[5 + k], r[k + 1].a); cfma(h.Bb, vB[5 + k], r[k + 1].b);
    }
}

template <bool FLUSH, bool REDUCE, bool DIAG, bool RX>
__global__ void __launch_bounds__(kThreads, 1) k_pair_sq(const TermParams p, const Geom g)
{
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t bars[2 * kMaxStages + 2 * kMaxRing];   // stage full | stage empty | ring full | ring empty
    __shared__ double red_s[REDUCE ? kMainW : 1][REDUCE ? kBT : 1][3];

    const int tid = threadIdx.x;
    const bool sub_y = p.flags & F_SUB_Y;                  // stage 1 subtracts T_{k-2}: always, except on the pair (1, 2)
    const bool need_acc = FLUSH && !(p.flags & F_ACC_INIT);
    const bool use_st = sub_y || DIAG;                     // the stage carries T_{k-2} and / or the diagonal
    const uint32_t stb = (uint32_t)g.stage_bytes;
    const int S = g.n_stage;
    const uint32_t NA = (uint32_t)g.n_ring;
    const uint32_t bar0 = smem_u32(bars), smem0 = smem_u32(smem);
    const uint32_t b_sfull = bar0, b_sempty = bar0 + 8 * kMaxStages, b_rfull = bar0 + 16 * kMaxStages, b_rempty = b_rfull + 8 * kMaxRing;
    const uint32_t ringA0 = smem0, ringB0 = ringA0 + NA * kSlotBytes, stage0 = ringB0 + kNB * kSlotBytes;

    if (tid == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(b_sfull + 8 * s, 1); mbar_init(b_sempty + 8 * s, kNW); }
        for (uint32_t s = 0; s < NA; ++s) { mbar_init(b_rfull + 8 * s, 1); mbar_init(b_rempty + 8 * s, kNW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // Runs: run u covers in-line position u % d0 of the lines [(u / d0) * len, ...); dealt to the blocks round-robin.
    const int64_t n_chunks = (g.n_lines + g.len - 1) / g.len;
    const int64_t n_runs = g.d0 * n_chunks;
    struct Run { int64_t line0, pos; int len; };
    auto run_of = [&](int64_t u) -> Run {
        Run r;
        const int64_t chunk = u / g.d0;
        r.pos = u - chunk * g.d0;
        r.line0 = chunk * g.len;
        r.len = (int)min((int64_t)g.len, g.n_lines - r.line0);
        return r;
    };
    auto wrap_line = [&](int64_t line) -> int64_t { return line < 0 ? line + g.n_lines : (line >= g.n_lines ? line - g.n_lines : line); };

    if (tid >= kConsumers) {
        // ------------------------------- producers: one thread of each of the two producer warps -------------------------------
        if ((tid & 31) != 0) return;
        // `halo` rows on either side of the tile's 128, taken round the periodic line
        auto load_rows = [&](uint32_t dst, const void *line_base_v, int64_t x0, int halo, uint32_t full, uint32_t rb = kRowBytes) {
            const char *line_base = static_cast<const char *>(line_base_v);   // rb = bytes per row (128: a vector row, 8: the diagonal)
            const bool wrap_lo = x0 == 0, wrap_hi = x0 + kR == g.W;
            const int lo = wrap_lo ? 0 : -halo, hi = wrap_hi ? kR : kR + halo;
            bulk_g2s(dst + (uint32_t)(lo + halo) * rb, line_base + (x0 + lo) * (int64_t)rb, (uint32_t)(hi - lo) * rb, full);
            if (wrap_lo) bulk_g2s(dst, line_base + (g.W - halo) * (int64_t)rb, (uint32_t)halo * rb, full);
            if (wrap_hi) bulk_g2s(dst + (uint32_t)(kR + halo) * rb, line_base, (uint32_t)halo * rb, full);
        };
        if (tid == kConsumers) {
            RingPos rp{0u, 1u};
            for (int64_t u = blockIdx.x; u < n_runs; u += gridDim.x) {
                const Run r = run_of(u);
                for (int j = -2; j < r.len + 2; ++j) {     // T_{k-1}: lines line0 - 2 .. line0 + len + 1, rows x0 - 2 .. x0 + 129
                    mbar_wait_idle(b_rempty + 8 * rp.i, rp.ph);
                    const uint32_t full = b_rfull + 8 * rp.i;
                    mbar_expect_tx(full, kSlotBytes);
                    load_rows(ringA0 + rp.i * kSlotBytes, p.x + wrap_line(r.line0 + j) * g.W * kBT, r.pos * kR, 2, full);
                    rp.adv(NA);
                }
            }
        } else if (use_st) {
            int s = 0;
            uint32_t sph = 1;
            for (int64_t u = blockIdx.x; u < n_runs; u += gridDim.x) {
                const Run r = run_of(u);
                for (int j = -1; j < r.len + 1; ++j) {     // T_{k-2}: lines line0 - 1 .. line0 + len, rows x0 - 1 .. x0 + 128
                    mbar_wait_idle(b_sempty + 8 * s, sph);
                    const uint32_t full = b_sfull + 8 * s;
                    mbar_expect_tx(full, (sub_y ? (uint32_t)kYBytes : 0u) + (DIAG ? (uint32_t)kDiagRows * 8u : 0u));
                    const int64_t line = wrap_line(r.line0 + j);
                    if (sub_y) load_rows(stage0 + (uint32_t)s * stb, p.y + line * g.W * kBT, r.pos * kR, 1, full);
                    if (DIAG) load_rows(stage0 + (uint32_t)s * stb + kYBytes, p.diag + line * g.W, r.pos * kR, 2, full, 8u);   // halo 2: 16-byte aligned
                    if (++s == S) { s = 0; sph ^= 1u; }
                }
            }
        }
        return;
    }

    // ---------------------------------------------------- consumer warps ----------------------------------------------------
    RingPos a0{0u, 0u}, a1{1u % NA, 0u}, a2{2u % NA, 0u};  // ring A loads holding the line above / the own line / the line below of stage 1
    int s = 0;
    uint32_t sph = 0;
    uint32_t it = 0;                                       // lines this block has taken: T_k of line `it` sits in ring B slot it % 4

    if (tid >= kMain) {
        // ---- halo warp: stage 1 for the two rows just outside the tile (tile rows -1 and 128), which stage 2 of the edge rows needs.
        // lane = (row, state, half of the eight directions); 4 complex FMAs per lane and line, the halves added by one shuffle.
        const int lane = tid & 31, hr = lane >> 4, state = (lane >> 1) & 7, dh = lane & 1;
        const uint32_t srow = hr ? (uint32_t)(kR + 2) : 1u;            // slot row of the halo row (slot row = tile row + 2)
        const uint32_t so = srow * kRowBytes + (uint32_t)state * 16u;
        // directions 0..7 = (line, in-line offset): (above, -1 0 +1), (own, -1 +1), (below, -1 0 +1)
        const int ln[4] = {dh ? 1 : 0, dh ? 2 : 0, dh ? 2 : 0, dh ? 2 : 1};
        const int dx[4] = {dh ? 1 : -1, dh ? -1 : 0, dh ? 0 : 1, dh ? 1 : -1};
        double2 hv[4];
#pragma unroll 1
        for (int64_t u = blockIdx.x; u < n_runs; u += gridDim.x) {
            const Run run = run_of(u);
            {
                int64_t x = run.pos * kR + (hr ? kR : -1);
                if (x < 0) x += g.W;
                if (x >= g.W) x -= g.W;
                const uint2 w = __ldg(reinterpret_cast<const uint2 *>(p.dline + x * kCH + dh * 4));
                const uint32_t id[4] = {w.x & 0xffffu, w.x >> 16, w.y & 0xffffu, w.y >> 16};
#pragma unroll
                for (int j = 0; j < 4; ++j) hv[j] = table_value(__ldg(p.vtab + (id[j] & 0x7fffu)), id[j]);
            }
#pragma unroll 1
            for (int i = 0; i < run.len + 2; ++i, ++it) {
                if (i == 0) {
                    mbar_wait(b_rfull + 8 * a0.i, a0.ph);
                    mbar_wait(b_rfull + 8 * a1.i, a1.ph);
                }
                mbar_wait(b_rfull + 8 * a2.i, a2.ph);
                if (use_st) mbar_wait(b_sfull + 8 * s, sph);
                const uint32_t sl[3] = {ringA0 + a0.i * kSlotBytes, ringA0 + a1.i * kSlotBytes, ringA0 + a2.i * kSlotBytes};
                double2 h = make_double2(0.0, 0.0);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    double2 xv;
                    lds_c(xv, (ln[j] == 0 ? sl[0] : ln[j] == 1 ? sl[1] : sl[2]) + so + (uint32_t)(dx[j] * kRowBytes));
                    cfma(h, hv[j], xv);
                }
                h.x += __shfl_xor_sync(0xffffffffu, h.x, 1);
                h.y += __shfl_xor_sync(0xffffffffu, h.y, 1);
                if (DIAG) {                                // + d * x on the halo row itself (diagonal stage index = tile row + 2)
                    double2 xo;
                    lds_c(xo, sl[1] + so);
                    const double d = lds_f64(stage0 + (uint32_t)s * stb + kYBytes + srow * 8u);
                    h.x = fma(d, xo.x, h.x); h.y = fma(d, xo.y, h.y);
                }
                h.x *= p.a; h.y *= p.a;
                if (sub_y) {                               // stage row = tile row + 1
                    double2 yv;
                    lds_c(yv, stage0 + (uint32_t)s * stb + (hr ? (uint32_t)(kR + 1) : 0u) * kRowBytes + (uint32_t)state * 16u);
                    h.x -= yv.x; h.y -= yv.y;
                }
                if (dh == 0) sts_c(ringB0 + (it % kNB) * kSlotBytes + so, h);
                const uint32_t rel = (uint32_t)__double2hiint(h.x) & (uint32_t)p.zero;
                asm volatile("bar.sync 1, %0;" ::"n"(kConsumers) : "memory");
                __syncwarp();
                if (lane == 0) {
                    if (use_st) mbar_arrive(b_sempty + 8 * s + rel);
                    mbar_arrive(b_rempty + 8 * a0.i + rel);
                    if (i == run.len + 1) { mbar_arrive(b_rempty + 8 * a1.i + rel); mbar_arrive(b_rempty + 8 * a2.i + rel); }
                }
                if (use_st) { if (++s == S) { s = 0; sph ^= 1u; } }
                a0.adv(NA); a1.adv(NA); a2.adv(NA);
            }
            a0.adv(NA); a0.adv(NA); a1.adv(NA); a1.adv(NA); a2.adv(NA); a2.adv(NA);
        }
        if (REDUCE) asm volatile("bar.sync 1, %0;" ::"n"(kConsumers) : "memory");   // the final reduction's barrier
        return;
    }

    // ---- main consumers: thread = states 2q, 2q + 1 of the tile rows A = 2 pr and B = 2 pr + 1 (pr = 0 .. 63), in both stages;
    // "slot a" of a thread is state 2q + par, "slot b" state 2q + 1 - par (conflict-free 128-bit accesses, term_sq.cu).
    const int pr = tid >> 2, q = tid & 3, par = pr & 1;
    const uint32_t oa = (uint32_t)(2 * q + par) * 16u, ob = (uint32_t)(2 * q + 1 - par) * 16u;
    const uint32_t rows2p = (uint32_t)(2 * pr + 1) * kRowBytes;  // 132-row slots: the slot row of tile row A - 1
    const uint32_t rowsy = (uint32_t)(2 * pr + 1) * kRowBytes;   // 130-row stage: the stage row of tile row A
    double2 vA[kCH], vB[kCH];                              // hopping values of the two rows by direction, kept for a whole run
    double sa_re = 0.0, sa_im = 0.0, sa_nn = 0.0, sb_re = 0.0, sb_im = 0.0, sb_nn = 0.0;
    Row2 partA, partB;                                     // cc*T_{k-1} + cd*T_{k-2} on the rows of the line that stage 2 takes next
    double dA = 0.0, dB = 0.0, dPA = 0.0, dPB = 0.0;       // DIAG: diagonal of rows A, B on stage 1's line / on stage 2's line (the line before)
    partA.a = partA.b = partB.a = partB.b = make_double2(0.0, 0.0);

#pragma unroll 1
    for (int64_t u = blockIdx.x; u < n_runs; u += gridDim.x) {
        const Run run = run_of(u);
        {   // the values of the thread's two rows: dline[x][direction] -> table entry (+ conjugate bit); the same on every line
            const int64_t xa = run.pos * kR + 2 * pr, xb = xa + 1;
            const uint4 ia = __ldg(reinterpret_cast<const uint4 *>(p.dline + xa * kCH));
            const uint4 ib = __ldg(reinterpret_cast<const uint4 *>(p.dline + xb * kCH));
            const uint32_t wa[4] = {ia.x, ia.y, ia.z, ia.w}, wb[4] = {ib.x, ib.y, ib.z, ib.w};
#pragma unroll
            for (int k = 0; k < kCH; ++k) {
                const uint32_t ida = (wa[k >> 1] >> ((k & 1) * 16)) & 0xffffu, idb = (wb[k >> 1] >> ((k & 1) * 16)) & 0xffffu;
                vA[k] = table_value(__ldg(p.vtab + (ida & 0x7fffu)), ida);
                vB[k] = table_value(__ldg(p.vtab + (idb & 0x7fffu)), idb);
            }
        }
        const int64_t rowA0 = run.pos * kR + 2 * pr;       // in-line position of row A
#pragma unroll 1
        for (int i = 0; i < run.len + 2; ++i, ++it) {
            // stage 1 takes line line0 - 1 + i (stored when it is one of the run's), stage 2 line line0 - 2 + i (when i >= 2)
            const bool st2 = i >= 2;
            if (DIAG) { dPA = dA; dPB = dB; }
            const int64_t e2A = ((run.line0 + i - 2) * g.W + rowA0) * kBT + 2 * q, e2B = e2A + kBT;
            // ---- stage 2's operands that are not staged (HBM latency: issue first)
            double2 aAa, aAb, aBa, aBb;                    // psi' on rows A, B in slot order
            aAa = aAb = aBa = aBb = make_double2(0.0, 0.0);
            double2 zAa, zAb, zBa, zBb;                    // psi0 on rows A, B in slot order (state 2q + par, 2q + 1 - par)
            if (FLUSH && st2 && need_acc) {                // 128-bit loads straight into slot order (no selects on arrival)
                aAa = __ldcs(p.acc + e2A + par); aAb = __ldcs(p.acc + e2A + (1 - par));
                aBa = __ldcs(p.acc + e2B + par); aBb = __ldcs(p.acc + e2B + (1 - par));
            }
            if (REDUCE && st2 && q == 0) { prefetch_l2(p.psi0 + e2A); prefetch_l2(p.psi0 + e2B); }   // loaded after stage 1: 8 registers less there
            if (i == 0) {
                mbar_wait(b_rfull + 8 * a0.i, a0.ph);
                mbar_wait(b_rfull + 8 * a1.i, a1.ph);
            }
            mbar_wait(b_rfull + 8 * a2.i, a2.ph);
            if (use_st) mbar_wait(b_sfull + 8 * s, sph);
            const uint32_t sa0 = ringA0 + a0.i * kSlotBytes + rows2p, sa1 = ringA0 + a1.i * kSlotBytes + rows2p,
                           sa2 = ringA0 + a2.i * kSlotBytes + rows2p, sy = stage0 + (uint32_t)s * stb + rowsy;
            uint32_t rel;
            {   // ---- stage 1: T_k = a1 * H * T_{k-1} - T_{k-2} on rows A, B of line line0 - 1 + i
                Out4 h;
                Row2 xA, xB;
                apply_h<RX>(sa0, sa1, sa2, oa, ob, vA, vB, h, xA, xB);
                if (DIAG) {                                // diagonal of rows A, B of this line (stage index = tile row + 2); kept for stage 2 of the next line
                    const uint32_t sd = stage0 + (uint32_t)s * stb + kYBytes + (uint32_t)(2 * pr + 2) * 8u;
                    dA = lds_f64(sd); dB = lds_f64(sd + 8u);
                    h.Aa.x = fma(dA, xA.a.x, h.Aa.x); h.Aa.y = fma(dA, xA.a.y, h.Aa.y); h.Ab.x = fma(dA, xA.b.x, h.Ab.x); h.Ab.y = fma(dA, xA.b.y, h.Ab.y);
                    h.Ba.x = fma(dB, xB.a.x, h.Ba.x); h.Ba.y = fma(dB, xB.a.y, h.Ba.y); h.Bb.x = fma(dB, xB.b.x, h.Bb.x); h.Bb.y = fma(dB, xB.b.y, h.Bb.y);
                }
                h.Aa.x *= p.a; h.Aa.y *= p.a; h.Ab.x *= p.a; h.Ab.y *= p.a; h.Ba.x *= p.a; h.Ba.y *= p.a; h.Bb.x *= p.a; h.Bb.y *= p.a;
                if (sub_y) {
                    Row2 yA, yB;
                    lds_c(yA.a, sy + oa); lds_c(yA.b, sy + ob); lds_c(yB.a, sy + kRowBytes + oa); lds_c(yB.b, sy + kRowBytes + ob);
                    h.Aa.x -= yA.a.x; h.Aa.y -= yA.a.y; h.Ab.x -= yA.b.x; h.Ab.y -= yA.b.y;
                    h.Ba.x -= yB.a.x; h.Ba.y -= yB.a.y; h.Bb.x -= yB.b.x; h.Bb.y -= yB.b.y;
                }
                rel = (uint32_t)(__double2hiint(h.Aa.x) ^ __double2hiint(h.Ab.x) ^ __double2hiint(h.Ba.x) ^ __double2hiint(h.Bb.x));
                if (DIAG) rel ^= (uint32_t)(__double2hiint(dA) ^ __double2hiint(dB));
                const uint32_t wb = ringB0 + (it % kNB) * kSlotBytes + rows2p + kRowBytes;   // slot rows 2p + 1, 2p + 2 = rows A, B
                sts_c(wb + oa, h.Aa); sts_c(wb + ob, h.Ab); sts_c(wb + kRowBytes + oa, h.Ba); sts_c(wb + kRowBytes + ob, h.Bb);
                if (!REDUCE && i >= 1 && i <= run.len) {   // T_k of the run's own lines: read by the next pair, a whole sweep later
                    const int64_t e1A = ((run.line0 + i - 1) * g.W + rowA0) * kBT + 2 * q;
                    CVec<2> out;
                    out.v[0] = par ? h.Ab : h.Aa; out.v[1] = par ? h.Aa : h.Ab; out.st_stream(p.out1 + e1A);
                    out.v[0] = par ? h.Bb : h.Ba; out.v[1] = par ? h.Ba : h.Bb; out.st_stream(p.out1 + e1A + kBT);
                }
            }
            asm volatile("bar.sync 1, %0;" ::"n"(kConsumers) : "memory");   // line `it` of T_k is complete in ring B
            if (REDUCE && st2) {   // four 128-bit loads straight into slot order: no selects that would wait for the data here (L2 hits)
                zAa = __ldcs(p.psi0 + e2A + par); zAb = __ldcs(p.psi0 + e2A + (1 - par));
                zBa = __ldcs(p.psi0 + e2B + par); zBb = __ldcs(p.psi0 + e2B + (1 - par));
            }
            if (st2) {
                // ---- stage 2: T_{k+1} = a2 * H * T_k - T_{k-1} on rows A, B of line line0 - 2 + i (T_k lines it - 2, it - 1, it)
                const uint32_t sb0 = ringB0 + ((it - 2) % kNB) * kSlotBytes + rows2p, sb1 = ringB0 + ((it - 1) % kNB) * kSlotBytes + rows2p,
                               sb2 = ringB0 + (it % kNB) * kSlotBytes + rows2p;
                Out4 h;
                Row2 tA, tB, xA, xB;                       // T_k and T_{k-1} on the own rows
                apply_h<RX>(sb0, sb1, sb2, oa, ob, vA, vB, h, tA, tB);
                if (DIAG) {
                    h.Aa.x = fma(dPA, tA.a.x, h.Aa.x); h.Aa.y = fma(dPA, tA.a.y, h.Aa.y); h.Ab.x = fma(dPA, tA.b.x, h.Ab.x); h.Ab.y = fma(dPA, tA.b.y, h.Ab.y);
                    h.Ba.x = fma(dPB, tB.a.x, h.Ba.x); h.Ba.y = fma(dPB, tB.a.y, h.Ba.y); h.Bb.x = fma(dPB, tB.b.x, h.Bb.x); h.Bb.y = fma(dPB, tB.b.y, h.Bb.y);
                }
                lds_c(xA.a, sa0 + kRowBytes + oa); lds_c(xA.b, sa0 + kRowBytes + ob);
                lds_c(xB.a, sa0 + 2 * kRowBytes + oa); lds_c(xB.b, sa0 + 2 * kRowBytes + ob);
                h.Aa.x = fma(p.a2, h.Aa.x, -xA.a.x); h.Aa.y = fma(p.a2, h.Aa.y, -xA.a.y); h.Ab.x = fma(p.a2, h.Ab.x, -xA.b.x); h.Ab.y = fma(p.a2, h.Ab.y, -xA.b.y);
                h.Ba.x = fma(p.a2, h.Ba.x, -xB.a.x); h.Ba.y = fma(p.a2, h.Ba.y, -xB.a.y); h.Bb.x = fma(p.a2, h.Bb.x, -xB.b.x); h.Bb.y = fma(p.a2, h.Bb.y, -xB.b.y);
                rel ^= (uint32_t)(__double2hiint(h.Aa.x) ^ __double2hiint(h.Ab.x) ^ __double2hiint(h.Ba.x) ^ __double2hiint(h.Bb.x));
                CVec<2> out;
                if (!REDUCE) {
                    out.v[0] = par ? h.Ab : h.Aa; out.v[1] = par ? h.Aa : h.Ab; out.st_stream(p.out2 + e2A);
                    out.v[0] = par ? h.Bb : h.Ba; out.v[1] = par ? h.Ba : h.Bb; out.st_stream(p.out2 + e2B);
                }
                if (FLUSH) {
                    aAa.x += partA.a.x; aAa.y += partA.a.y; aAb.x += partA.b.x; aAb.y += partA.b.y;
                    aBa.x += partB.a.x; aBa.y += partB.a.y; aBb.x += partB.b.x; aBb.y += partB.b.y;
                    cfma(aAa, p.cb, tA.a); cfma(aAb, p.cb, tA.b); cfma(aBa, p.cb, tB.a); cfma(aBb, p.cb, tB.b);
                    cfma(aAa, p.ca, h.Aa); cfma(aAb, p.ca, h.Ab); cfma(aBa, p.ca, h.Ba); cfma(aBb, p.ca, h.Bb);
                    CVec<2> oA, oB;
                    oA.v[0] = par ? aAb : aAa; oA.v[1] = par ? aAa : aAb;
                    oB.v[0] = par ? aBb : aBa; oB.v[1] = par ? aBa : aBb;
                    if (REDUCE) {
                        auto acc3 = [](double &re, double &im, double &nn, double2 z, double2 v) {
                            re = fma(z.x, v.x, re); re = fma(z.y, v.y, re);
                            im = fma(z.x, v.y, im); im = fma(-z.y, v.x, im);
                            nn = fma(v.x, v.x, nn); nn = fma(v.y, v.y, nn);
                        };
                        acc3(sa_re, sa_im, sa_nn, zAa, aAa); acc3(sb_re, sb_im, sb_nn, zAb, aAb); oA.st(p.acc + e2A);
                        acc3(sa_re, sa_im, sa_nn, zBa, aBa); acc3(sb_re, sb_im, sb_nn, zBb, aBb); oB.st(p.acc + e2B);
                    } else {
                        oA.st_stream(p.acc + e2A);
                        oB.st_stream(p.acc + e2B);
                    }
                }
            }
            if (FLUSH) {   // the part of psi' that stage 2 cannot reach a line later: cc*T_{k-1} + cd*T_{k-2} on rows A, B of stage 1's line
                Row2 xA, xB;
                lds_c(xA.a, sa1 + kRowBytes + oa); lds_c(xA.b, sa1 + kRowBytes + ob);
                lds_c(xB.a, sa1 + 2 * kRowBytes + oa); lds_c(xB.b, sa1 + 2 * kRowBytes + ob);
                partA.a = partA.b = partB.a = partB.b = make_double2(0.0, 0.0);
                cfma(partA.a, p.cc, xA.a); cfma(partA.b, p.cc, xA.b); cfma(partB.a, p.cc, xB.a); cfma(partB.b, p.cc, xB.b);
                if (sub_y) {
                    Row2 yA, yB;
                    lds_c(yA.a, sy + oa); lds_c(yA.b, sy + ob); lds_c(yB.a, sy + kRowBytes + oa); lds_c(yB.b, sy + kRowBytes + ob);
                    cfma(partA.a, p.cd, yA.a); cfma(partA.b, p.cd, yA.b); cfma(partB.a, p.cd, yB.a); cfma(partB.b, p.cd, yB.b);
                }
                rel ^= (uint32_t)(__double2hiint(partA.a.x) ^ __double2hiint(partA.b.x) ^ __double2hiint(partB.a.x) ^ __double2hiint(partB.b.x));
            }
            // Every shared-memory read of this line must have RETURNED before the stage and the oldest ring slot are handed back:
            // the barrier addresses depend on the registers they filled (`rel` is 0: p.zero is 0, but only at run time).
            rel &= (uint32_t)p.zero;
            __syncwarp();
            if ((tid & 31) == 0) {
                if (use_st) mbar_arrive(b_sempty + 8 * s + rel);
                mbar_arrive(b_rempty + 8 * a0.i + rel);
                if (i == run.len + 1) { mbar_arrive(b_rempty + 8 * a1.i + rel); mbar_arrive(b_rempty + 8 * a2.i + rel); }
            }
            if (use_st) { if (++s == S) { s = 0; sph ^= 1u; } }
            a0.adv(NA); a1.adv(NA); a2.adv(NA);
        }
        a0.adv(NA); a0.adv(NA); a1.adv(NA); a1.adv(NA); a2.adv(NA); a2.adv(NA);   // len + 2 lines consume len + 4 ring loads
    }

    if (REDUCE) {
        double s_re[2] = {par ? sb_re : sa_re, par ? sa_re : sb_re};   // state order 2q, 2q + 1
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
        asm volatile("bar.sync 1, %0;" ::"n"(kConsumers) : "memory");   // consumers only (the producer warps have left)
        if (tid < kBT * 3) {
            const int bb = tid / 3, c = tid % 3;
            double t = 0.0;
#pragma unroll
            for (int w2 = 0; w2 < kMainW; ++w2) t += red_s[w2][bb][c];
            p.partial[((int64_t)blockIdx.x * kBT + bb) * 3 + c] = t;
        }
    }
}

bool make_geom(const TermParams &p, Geom &g)
{
    if (p.sq8_line <= 0 || !p.dline || !p.uniform || p.max_row_off != kCH || p.n_table <= 1 || p.packed) return false;
    const int64_t W = p.sq8_line;
    if (W % kR != 0 || p.n_orb % W != 0 || p.n_orb / W < 4 || p.n_orb >= ((int64_t)1 << 31)) return false;
    g.W = W; g.d0 = W / kR; g.n_lines = p.n_orb / W;
    g.len = (int)std::min<int64_t>(std::max(1, knob("sq2_len", 64)), g.n_lines);
    // Less is more: every KB of shared memory is a KB less of L1 for the streamed stores and the psi' loads in flight
    // (cfg4: 1080 us per term with 5 + 3 slots, 1009 with 4 + 3, 1016 with 5 + 2).
    g.n_ring = std::min(kMaxRing, std::max(4, knob("sq2_ring", 4)));
    g.n_stage = std::min(kMaxStages, std::max(2, knob("sq2_stages", 3)));
    g.stage_bytes = kYBytes + (p.diag ? kDiagBytes : 0);
    return (size_t)(g.n_ring + kNB) * kSlotBytes + (size_t)g.n_stage * g.stage_bytes <= kSmemMax - 4096;
}

template <bool FLUSH, bool REDUCE, bool DIAG, bool RX>
int launch_one(const TermParams &p, const Geom &g, int num_sms, cudaStream_t st, int *grid_out)
{
    const size_t dyn = (size_t)(g.n_ring + kNB) * kSlotBytes + (size_t)g.n_stage * g.stage_bytes;
    auto kern = k_pair_sq<FLUSH, REDUCE, DIAG, RX>;
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

}  // namespace sq2

// Tiles of 8 states on the square lattice that term_sq.cu runs on (with or without a real diagonal).
bool pair_sq_supported(int bt, const TermParams &p)
{
    if (bt != sq2::kBT || !knob("sq2", 1)) return false;
    sq2::Geom g;
    return sq2::make_geom(p, g);
}

// p.x = T_{k-1}, p.y = T_{k-2} (read only), p.out1 <- T_k, p.out2 <- T_{k+1} (neither is stored with F_REDUCE), p.a / p.a2 the two
// scale factors, p.n_acc > 0: psi' (p.acc) += ca*T_{k+1} + cb*T_k + cc*T_{k-1} + cd*T_{k-2} (F_ACC_INIT: psi' = ...), F_SUB_Y: T_{k-2}
// exists (k >= 2), F_REDUCE: the dot products of the last pair (implies n_acc > 0).
int launch_pair_sq(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    sq2::Geom g;
    if (!sq2::make_geom(p, g) || !p.out1 || !p.out2) return TBPM_EINVAL;
    const bool red = p.flags & F_REDUCE;
    if (red && p.n_acc <= 0) return TBPM_EINVAL;
    const int shape = red ? 2 : (p.n_acc > 0 ? 1 : 0);    // plain pair / pair with psi' update / last pair
#define TBPM_PAIR(D, R)                                                                                         \
    (shape == 2 ? sq2::launch_one<true, true, D, R>(p, g, num_sms, st, grid_out)                                  \
                : shape == 1 ? sq2::launch_one<true, false, D, R>(p, g, num_sms, st, grid_out) : sq2::launch_one<false, false, D, R>(p, g, num_sms, st, grid_out))
    if (p.diag) return p.sq8_real_x ? TBPM_PAIR(true, true) : TBPM_PAIR(true, false);
    return p.sq8_real_x ? TBPM_PAIR(false, true) : TBPM_PAIR(false, false);
#undef TBPM_PAIR
}

}  // namespace tbpm_detail

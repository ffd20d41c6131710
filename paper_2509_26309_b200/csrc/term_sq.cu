// term_sq.cu -- fused Chebyshev term on the PERIODIC SQUARE LATTICE WITH NEXT-NEAREST NEIGHBOURS (offsets {-W-1, -W, -W+1, -1, +1,
// W-1, W, W+1}) whose complex hopping values depend on the position ALONG the line only -- Peierls phases in the Landau gauge,
// BASELINE.json:configs[3].  Tiles of 8 interleaved states.
//
//   T_k = a*H*T_{k-1} - T_{k-2}  (amxsy) + deferred psi' accumulation (axpy) + last-term
//   <psi0|psi'>, <psi'|psi'> (calc_corr_dos), exactly as term_ph.cuh; same TermParams, same results.
//
// Why (profiles/r2_ncu_cfg4.md): on this lattice the rolling-window kernel (term_rw.cu) is bound by the L1 data pipe and by
// instruction issue, not by the HBM: per row it reads 8 column words, 8 value indices and 8 table values on top of the vector
// rows, compares the columns with the lattice, and swaps state halves.  The builder (build.cu, k_sq8) has verified for EVERY row
// that its columns are its eight periodic neighbours and that the value in direction k is table[dline[x][k]], so here
//   matrix  nothing is read per row: a block walks along W (down the lattice) at a fixed in-line position, and every thread
//           fetches the 2 x 8 hopping values of its two rows ONCE per run of 64 tiles (dline + value table) into registers;
//   ring    n_ring slots of 128 + 2 rows of x, one bulk copy (TMA) per tile; the rows beyond the ends of a line and the lines
//           beyond the ends of the lattice are the WRAPPED ones, so seam rows are like all others;
//   stage   the tile's 128 rows of y (T_{k-2}) (and of the diagonal, if any), n_stage tiles ahead;
//   consumers  8 warps; thread = 2 states of two ADJACENT rows: the 4 rows r-1 .. r+2 of each of the three lines are read once
//           and serve both rows (12 row reads for 16 neighbours), the two rows' state halves are read in opposite order by
//           neighbouring row pairs (conflict-free LDS.128); 320 threads leave every thread ~160 registers for the 64 that
//           hold the values.
// Per row and state tile this is 100 instructions instead of 360, and 900 instead of 1,850 bytes through the L1 data pipe.
#include <algorithm>

#include "term_ph.cuh"

namespace tbpm_detail {
namespace sq {

using namespace ph;

constexpr int kBT = 8, kNW = 8, kConsumers = kNW * 32, kThreads = kConsumers + 64;
constexpr int kR = 128;                                    // rows per tile: 64 row pairs x 4 lanes
constexpr int kRowBytes = kBT * 16;
constexpr int kSlotBytes = (kR + 2) * kRowBytes;           // 16,640
constexpr int kMaxRing = 8;
constexpr int kCH = 8;

struct Geom {
    int64_t W;                  // rows per lattice line
    int64_t d0;                 // tiles per line
    int64_t n_lines;
    int len;                    // lines per run
    int n_ring, n_stage;
    int off_y, off_diag, stage_bytes;
};

struct RingPos {
    uint32_t i, ph;
    __device__ __forceinline__ void adv(uint32_t nr) { if (++i == nr) { i = 0; ph ^= 1u; } }
};

__device__ __forceinline__ void lds_c(double2 &v, uint32_t a)
{
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
}

struct Row2 { double2 a, b; };                             // the thread's two states of one row (slot a / slot b, see `par`)

template <int NACC, bool REDUCE>
__global__ void __launch_bounds__(kThreads, 1) k_term_sq(const TermParams p, const Geom g)
{
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t bars[2 * kMaxStages + 2 * kMaxRing];   // stage full | stage empty | ring full | ring empty
    __shared__ double red_s[REDUCE ? kNW : 1][REDUCE ? kBT : 1][3];

    const int tid = threadIdx.x;
    const bool sub_y = p.flags & F_SUB_Y;
    const bool need_y = sub_y || NACC == 3;
    const bool need_acc = NACC > 0 && !(p.flags & F_ACC_INIT);
    const bool has_diag = p.diag != nullptr;
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

    if (tid >= kConsumers) {
        // ------------------------------- producers: one thread of each of the two producer warps -------------------------------
        if ((tid & 31) != 0) return;
        if (tid == kConsumers) {
            RingPos rp{0u, 1u};
            // rows [pos * 128 - 1, pos * 128 + 129) of a line; the line index and the two end rows wrap round the periodic lattice
            auto ring_load = [&](int64_t line, int64_t pos) {
                mbar_wait(b_rempty + 8 * rp.i, rp.ph);
                const uint32_t full = b_rfull + 8 * rp.i, slot = ring0 + rp.i * kSlotBytes;
                if (line < 0) line += g.n_lines;
                if (line >= g.n_lines) line -= g.n_lines;
                const double2 *base = p.x + line * g.W * kBT;
                const int64_t x0 = pos * kR;
                const bool wrap_lo = x0 == 0, wrap_hi = x0 + kR == g.W;
                const int lo = wrap_lo ? 0 : -1, hi = wrap_hi ? kR : kR + 1;
                mbar_expect_tx(full, kSlotBytes);
                bulk_g2s(slot + (uint32_t)(lo + 1) * kRowBytes, base + (x0 + lo) * kBT, (uint32_t)(hi - lo) * kRowBytes, full);
                if (wrap_lo) bulk_g2s(slot, base + (g.W - 1) * kBT, kRowBytes, full);
                if (wrap_hi) bulk_g2s(slot + (uint32_t)(kR + 1) * kRowBytes, base, kRowBytes, full);
                rp.adv(NR);
            };
            for (int64_t u = blockIdx.x; u < n_runs; u += gridDim.x) {
                const Run r = run_of(u);
                ring_load(r.line0 - 1, r.pos);
                ring_load(r.line0, r.pos);
                for (int j = 0; j < r.len; ++j) ring_load(r.line0 + j + 1, r.pos);
            }
        } else {
            int s = 0;
            uint32_t sph = 1;
            const uint32_t tx = (need_y ? kR * kRowBytes : 0u) + (has_diag ? kR * 8u : 0u);
            for (int64_t u = blockIdx.x; u < n_runs; u += gridDim.x) {
                const Run r = run_of(u);
                for (int j = 0; j < r.len; ++j) {
                    const int64_t r0 = (r.line0 + j) * g.W + r.pos * kR;
                    mbar_wait(b_sempty + 8 * s, sph);
                    const uint32_t full = b_sfull + 8 * s, st = stage0 + (uint32_t)s * (uint32_t)g.stage_bytes;
                    mbar_expect_tx(full, tx);
                    if (need_y) bulk_g2s(st + g.off_y, p.y + r0 * kBT, kR * kRowBytes, full);
                    if (has_diag) bulk_g2s(st + g.off_diag, p.diag + r0, kR * 8, full);
                    if (++s == S) { s = 0; sph ^= 1u; }
                }
            }
        }
        return;
    }

    // ---------------------------------------------------- consumer warps ----------------------------------------------------
    // thread = states 2q, 2q + 1 of the tile rows A = 2 pr and B = 2 pr + 1.  Neighbouring row pairs read the two 16-byte halves
    // in opposite order (par), so that a quarter-warp (2 pairs x 4 lanes) touches all 32 banks: "slot a" of a thread is state
    // 2q + par, "slot b" state 2q + 1 - par.
    const int pr = tid >> 2, q = tid & 3, par = pr & 1;
    const uint32_t oa = (uint32_t)(2 * q + par) * 16u, ob = (uint32_t)(2 * q + 1 - par) * 16u;
    const uint32_t rowsA = (uint32_t)(2 * pr) * kRowBytes;             // slot row index of tile row A - 1 (the slot starts with the halo row)
    const uint32_t yoff = (uint32_t)(2 * pr) * kRowBytes;
    double2 vA[kCH], vB[kCH];                                          // hopping values of the two rows by direction, kept for a whole run
    double sa_re = 0.0, sa_im = 0.0, sa_nn = 0.0, sb_re = 0.0, sb_im = 0.0, sb_nn = 0.0;

    RingPos r0p{0u, 0u}, r1p{1u % NR, 0u}, r2p{2u % NR, 0u};           // ring loads holding the line above / the own line / the line below
    int s = 0;
    uint32_t sph = 0, st = stage0;

    auto load4 = [&](uint32_t base, Row2 (&r)[4]) {                    // rows A - 1, A, B, B + 1 of one line
#pragma unroll
        for (int i = 0; i < 4; ++i) { lds_c(r[i].a, base + (uint32_t)i * kRowBytes + oa); lds_c(r[i].b, base + (uint32_t)i * kRowBytes + ob); }
    };

#pragma unroll 1
    for (int64_t u = blockIdx.x; u < n_runs; u += gridDim.x) {
        const Run run = run_of(u);
        {   // the values of the thread's two rows: dline[x][direction] -> table entry (+ conjugate bit); the same on every line
            const int64_t x = run.pos * kR + 2 * pr;
            const uint4 ia = __ldg(reinterpret_cast<const uint4 *>(p.dline + x * kCH));
            const uint4 ib = __ldg(reinterpret_cast<const uint4 *>(p.dline + (x + 1) * kCH));
            const uint32_t wa[4] = {ia.x, ia.y, ia.z, ia.w}, wb[4] = {ib.x, ib.y, ib.z, ib.w};
#pragma unroll
            for (int k = 0; k < kCH; ++k) {
                const uint32_t ida = (wa[k >> 1] >> ((k & 1) * 16)) & 0xffffu, idb = (wb[k >> 1] >> ((k & 1) * 16)) & 0xffffu;
                vA[k] = table_value(__ldg(p.vtab + (ida & 0x7fffu)), ida);
                vB[k] = table_value(__ldg(p.vtab + (idb & 0x7fffu)), idb);
            }
        }
        int64_t row0 = run.line0 * g.W + run.pos * kR;
#pragma unroll 1
        for (int j = 0; j < run.len; ++j, row0 += g.W) {
            const int64_t eA = (row0 + 2 * pr) * kBT + 2 * q, eB = eA + kBT;
            // ---- operands that are not staged (HBM latency: issue first)
            CVec<2> aoldA, aoldB, zA, zB;
            if (NACC > 0) { aoldA.stream_if(p.acc + eA, need_acc); aoldB.stream_if(p.acc + eB, need_acc); }
            if (REDUCE) { zA.stream_if(p.psi0 + eA, true); zB.stream_if(p.psi0 + eB, true); }
            if (j == 0) {
                mbar_wait(b_rfull + 8 * r0p.i, r0p.ph);
                mbar_wait(b_rfull + 8 * r1p.i, r1p.ph);
            }
            mbar_wait(b_rfull + 8 * r2p.i, r2p.ph);
            mbar_wait(b_sfull + 8 * s, sph);
            const uint32_t bp = ring0 + r0p.i * kSlotBytes + rowsA, bo = ring0 + r1p.i * kSlotBytes + rowsA, bn = ring0 + r2p.i * kSlotBytes + rowsA;
            double2 hAa = make_double2(0.0, 0.0), hAb = hAa, hBa = hAa, hBb = hAa;
            Row2 r[4];
            load4(bp, r);                                              // line above: directions 0, 1, 2 = in-line offsets -1, 0, +1
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                cfma(hAa, vA[k], r[k].a); cfma(hAb, vA[k], r[k].b);
                cfma(hBa, vB[k], r[k + 1].a); cfma(hBb, vB[k], r[k + 1].b);
            }
            load4(bo, r);                                              // own line: directions 3, 4 = -1, +1; r[1], r[2] are x[A], x[B]
            cfma(hAa, vA[3], r[0].a); cfma(hAb, vA[3], r[0].b);
            cfma(hBa, vB[3], r[1].a); cfma(hBb, vB[3], r[1].b);
            cfma(hAa, vA[4], r[2].a); cfma(hAb, vA[4], r[2].b);
            cfma(hBa, vB[4], r[3].a); cfma(hBb, vB[4], r[3].b);
            const Row2 xA = r[1], xB = r[2];
            load4(bn, r);                                              // line below: directions 5, 6, 7
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                cfma(hAa, vA[5 + k], r[k].a); cfma(hAb, vA[5 + k], r[k].b);
                cfma(hBa, vB[5 + k], r[k + 1].a); cfma(hBb, vB[5 + k], r[k + 1].b);
            }
            Row2 yA, yB;
            yA.a = yA.b = yB.a = yB.b = make_double2(0.0, 0.0);
            if (need_y) {
                lds_c(yA.a, st + g.off_y + yoff + oa); lds_c(yA.b, st + g.off_y + yoff + ob);
                lds_c(yB.a, st + g.off_y + yoff + kRowBytes + oa); lds_c(yB.b, st + g.off_y + yoff + kRowBytes + ob);
            }
            double dA = 0.0, dB = 0.0;
            if (has_diag) { dA = lds_f64(st + g.off_diag + (uint32_t)(2 * pr) * 8u); dB = lds_f64(st + g.off_diag + (uint32_t)(2 * pr + 1) * 8u); }
            if (has_diag) {
                hAa.x = fma(dA, xA.a.x, hAa.x); hAa.y = fma(dA, xA.a.y, hAa.y); hAb.x = fma(dA, xA.b.x, hAb.x); hAb.y = fma(dA, xA.b.y, hAb.y);
                hBa.x = fma(dB, xB.a.x, hBa.x); hBa.y = fma(dB, xB.a.y, hBa.y); hBb.x = fma(dB, xB.b.x, hBb.x); hBb.y = fma(dB, xB.b.y, hBb.y);
            }
            hAa.x *= p.a; hAa.y *= p.a; hAb.x *= p.a; hAb.y *= p.a; hBa.x *= p.a; hBa.y *= p.a; hBb.x *= p.a; hBb.y *= p.a;
            if (sub_y) {
                hAa.x -= yA.a.x; hAa.y -= yA.a.y; hAb.x -= yA.b.x; hAb.y -= yA.b.y;
                hBa.x -= yB.a.x; hBa.y -= yB.a.y; hBb.x -= yB.b.x; hBb.y -= yB.b.y;
            }
            // Every shared-memory read of this tile must have RETURNED before the stage and the oldest ring slot are handed back:
            // the barrier addresses depend on the registers they filled (`rel` is 0: p.zero is 0, but only at run time).
            const uint32_t rel = (uint32_t)(__double2hiint(hAa.x) ^ __double2hiint(hAb.x) ^ __double2hiint(hBa.x) ^ __double2hiint(hBb.x) ^
                                            __double2hiint(yA.a.x) ^ __double2hiint(yA.b.x) ^ __double2hiint(yB.a.x) ^ __double2hiint(yB.b.x) ^
                                            __double2hiint(xA.a.x) ^ __double2hiint(xA.b.x) ^ __double2hiint(xB.a.x) ^ __double2hiint(xB.b.x) ^
                                            __double2hiint(dA) ^ __double2hiint(dB)) & (uint32_t)p.zero;
            __syncwarp();
            if ((tid & 31) == 0) {
                mbar_arrive(b_sempty + 8 * s + rel);
                mbar_arrive(b_rempty + 8 * r0p.i + rel);
                if (j == run.len - 1) { mbar_arrive(b_rempty + 8 * r1p.i + rel); mbar_arrive(b_rempty + 8 * r2p.i + rel); }
            }
            if (++s == S) { s = 0; sph ^= 1u; st = stage0; } else st += (uint32_t)g.stage_bytes;
            r0p.adv(NR); r1p.adv(NR); r2p.adv(NR);

            CVec<2> out;
            if (!REDUCE) {                                             // T_k: its readers come a whole sweep later
                out.v[0] = par ? hAb : hAa; out.v[1] = par ? hAa : hAb; out.st_stream(p.y + eA);
                out.v[0] = par ? hBb : hBa; out.v[1] = par ? hBa : hBb; out.st_stream(p.y + eB);
            }
            if (NACC > 0) {
                double2 aAa = par ? aoldA.v[1] : aoldA.v[0], aAb = par ? aoldA.v[0] : aoldA.v[1];
                double2 aBa = par ? aoldB.v[1] : aoldB.v[0], aBb = par ? aoldB.v[0] : aoldB.v[1];
                cfma(aAa, p.ca, hAa); cfma(aAb, p.ca, hAb); cfma(aBa, p.ca, hBa); cfma(aBb, p.ca, hBb);
                if (NACC >= 2) { cfma(aAa, p.cb, xA.a); cfma(aAb, p.cb, xA.b); cfma(aBa, p.cb, xB.a); cfma(aBb, p.cb, xB.b); }
                if (NACC == 3) { cfma(aAa, p.cc, yA.a); cfma(aAb, p.cc, yA.b); cfma(aBa, p.cc, yB.a); cfma(aBb, p.cc, yB.b); }
                CVec<2> oA, oB;
                oA.v[0] = par ? aAb : aAa; oA.v[1] = par ? aAa : aAb;
                oB.v[0] = par ? aBb : aBa; oB.v[1] = par ? aBa : aBb;
                if (REDUCE) {
                    const double2 zAa = par ? zA.v[1] : zA.v[0], zAb = par ? zA.v[0] : zA.v[1];
                    const double2 zBa = par ? zB.v[1] : zB.v[0], zBb = par ? zB.v[0] : zB.v[1];
                    auto acc3 = [](double &re, double &im, double &nn, double2 z, double2 v) {
                        re = fma(z.x, v.x, re); re = fma(z.y, v.y, re);
                        im = fma(z.x, v.y, im); im = fma(-z.y, v.x, im);
                        nn = fma(v.x, v.x, nn); nn = fma(v.y, v.y, nn);
                    };
                    acc3(sa_re, sa_im, sa_nn, zAa, aAa); acc3(sb_re, sb_im, sb_nn, zAb, aAb);
                    acc3(sa_re, sa_im, sa_nn, zBa, aBa); acc3(sb_re, sb_im, sb_nn, zBb, aBb);
                    oA.st(p.acc + eA); oB.st(p.acc + eB);              // psi': T_0 of the next step
                } else {
                    oA.st_stream(p.acc + eA); oB.st_stream(p.acc + eB);
                }
            }
        }
        r0p.adv(NR); r0p.adv(NR); r1p.adv(NR); r1p.adv(NR); r2p.adv(NR); r2p.adv(NR);   // a run of len tiles consumes len + 2 ring loads
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
            for (int w2 = 0; w2 < kNW; ++w2) t += red_s[w2][bb][c];
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
    g.len = (int)std::min<int64_t>(std::max(1, knob("sq_len", 64)), g.n_lines);
    size_t o = 0;
    g.off_y = (int)o;    o += (size_t)kR * kRowBytes;
    g.off_diag = (int)o; o += (size_t)kR * 8;
    g.stage_bytes = (int)((o + 127) & ~size_t(127));
    g.n_ring = std::min(kMaxRing, std::max(4, knob("sq_ring", 6)));
    g.n_stage = std::min(kMaxStages, std::max(2, knob("sq_stages", 4)));
    return (size_t)g.n_ring * kSlotBytes + (size_t)g.n_stage * g.stage_bytes <= kSmemMax - 4096;
}

template <int NACC, bool REDUCE>
int launch_one(const TermParams &p, const Geom &g, int num_sms, cudaStream_t st, int *grid_out)
{
    const size_t dyn = (size_t)g.n_ring * kSlotBytes + (size_t)g.n_stage * g.stage_bytes;
    auto kern = k_term_sq<NACC, REDUCE>;
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

}  // namespace sq

bool term_sq_supported(int bt, const TermParams &p)
{
    if (bt != sq::kBT || (p.flags & F_SKIP_H) || !knob("sq", 1)) return false;
    const bool red = p.flags & F_REDUCE, wy = p.flags & F_WRITE_Y;
    if (red == wy) return false;
    if (!red && !(p.n_acc == 0 || p.n_acc == 3)) return false;
    if (red && (p.n_acc < 1 || p.n_acc > 3)) return false;
    sq::Geom g;
    return sq::make_geom(p, g);
}

int launch_term_sq(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    sq::Geom g;
    if (!sq::make_geom(p, g)) return TBPM_EINVAL;
    const bool red = p.flags & F_REDUCE;
    if (!red && p.n_acc == 0) return sq::launch_one<0, false>(p, g, num_sms, st, grid_out);
    if (!red && p.n_acc == 3) return sq::launch_one<3, false>(p, g, num_sms, st, grid_out);
    if (red && p.n_acc == 1) return sq::launch_one<1, true>(p, g, num_sms, st, grid_out);
    if (red && p.n_acc == 2) return sq::launch_one<2, true>(p, g, num_sms, st, grid_out);
    if (red && p.n_acc == 3) return sq::launch_one<3, true>(p, g, num_sms, st, grid_out);
    return TBPM_EINVAL;
}

}  // namespace tbpm_detail

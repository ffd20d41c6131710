// term_l3.cu -- fused Chebyshev term on THREE-DIMENSIONAL LATTICES (offsets {+-1, +-S1, +-S2}, one real hopping value, optional
// real diagonal: the simple cubic lattice of BASELINE.json:configs[4] and its anisotropic relatives).  Tiles of 8 interleaved states.
//
//   T_k = a*H*T_{k-1} - T_{k-2}  (amxsy) + deferred psi' accumulation (axpy) + last-term
//   <psi0|psi'>, <psi'|psi'> (calc_corr_dos), exactly as term_ph.cuh; same TermParams, same results.
//
// Why (profiles/r2_ncu_cfg5.md): with 8 states a vector row is one 128-byte line.  The phased kernel asks the L1 for nine lines
// per row, the rolling-window kernel (term_rw.cu, one-dimensional tiles) still fetched the two in-plane line neighbours with LDG,
// and every LDG in flight needs a line of an L1 that the shared-memory ring has shrunk to a few dozen KB.  Here NOTHING of x is
// gathered through the L1:
//   tile   kTY = 4 line segments of kTX = 32 consecutive rows (128 rows), at the same position of consecutive planes;
//   ring   n_ring slots, one per plane: (kTY + 2) segments of kTX + 2 rows -- the tile's rows plus a one-row / one-line halo --
//          brought in by six bulk copies (TMA, SASS UBLKCP) of 4,352 bytes.  A block WALKS along S2 (the plane stride): the slot
//          loaded as "plane z + 1" serves tile z + 1 as its own rows and tile z + 2 as "plane z - 1", so every row of x enters the
//          SM 1.6 times (204 / 128) instead of three to nine times, all of it without a register or an L1 line held in flight;
//   stage  per tile: its 128 rows of y (T_{k-2}) and of the real diagonal, n_stage tiles ahead;
//   consumers (16 warps; thread = one state of two rows, so that eight lanes read one 128-byte row: conflict-free LDS.128, natural
//          state order, fully coalesced 128-bit stores) read the six neighbours, x[row] and y from shared memory.
// The column words are NOT read for rows whose entries sit exactly where the lattice puts them (one bit per row, written by
// build.cu's k_lat_flags); a warp pass that holds any other row (periodic seams, or a matrix that merely resembles a lattice)
// gathers its rows entry by entry from global memory through ocol -- always correct, only slower.  psi' and psi0 (every third
// term / last term only) are streamed with LDG as in term_ph.cuh.  Two producer threads (ring, stages) in warps of their own.
#include <algorithm>

#include "term_ph.cuh"

namespace tbpm_detail {
namespace l3 {

using namespace ph;

constexpr int kBT = 8, kNW = 16, kConsumers = kNW * 32, kThreads = kConsumers + 64;
constexpr int kTX = 32, kTY = 4, kR = kTX * kTY;            // 128 rows per tile
constexpr int kSegRows = kTX + 2, kSegs = kTY + 2;          // with halo
constexpr int kRowBytes = kBT * 16;
constexpr int kSegBytes = kSegRows * kRowBytes;             // 4,352
constexpr int kSlotBytes = kSegs * kSegBytes;               // 26,112
constexpr int kMaxRing = 6;
constexpr int kCH = 6;

struct Geom {
    int64_t S1, S2;             // line and plane stride in rows
    int64_t n_planes;           // n_orb / S2
    int nxg, nyg;               // tiles per line (S1 / kTX), tile rows per plane (S2 / S1 / kTY)
    int64_t n_pos;              // nxg * nyg: tile positions of a plane
    int len;                    // planes per run
    int n_ring, n_stage;
    int off_y, off_diag, stage_bytes;
};

struct RingPos {                                            // slot and barrier parity of one ring load, advanced incrementally
    uint32_t i, ph;
    __device__ __forceinline__ void adv(uint32_t nr) { if (++i == nr) { i = 0; ph ^= 1u; } }
};

__device__ __forceinline__ void lds_c(double2 &v, uint32_t a)
{
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
}
__device__ __forceinline__ double2 ldg_c(const double2 *p)
{
    double2 v;
    asm volatile("ld.global.nc.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ double2 ldg_stream_if(const double2 *p, bool on)      // read once: no L1 line, first out of L2; zero when off
{
    double2 v;
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %3, 0;\nmov.f64 %0, 0d0000000000000000;\nmov.f64 %1, 0d0000000000000000;\n"
                 "@q ld.global.cs.v2.f64 {%0, %1}, [%2];\n}"
                 : "=d"(v.x), "=d"(v.y)
                 : "l"(p), "r"((int)on)
                 : "memory");
    return v;
}
__device__ __forceinline__ void stg_stream(double2 *p, double2 v)
{
    asm volatile("st.global.cs.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ void stg(double2 *p, double2 v)
{
    asm volatile("st.global.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}

template <int NACC, bool REDUCE>
__global__ void __launch_bounds__(kThreads, 1) k_term_l3(const TermParams p, const Geom g)
{
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

    // Runs: run u covers tile position u % n_pos of the planes [(u / n_pos) * len, ...); dealt to the blocks round-robin, so the
    // blocks sweep neighbouring positions of the same planes together (the halos they share are L2 hits).
    const int64_t n_chunks = (g.n_planes + g.len - 1) / g.len;
    const int64_t n_runs = g.n_pos * n_chunks;
    struct Run { int64_t plane0, yg, xg, row0; int len; };   // first plane, tile row and tile column, first row of the first tile
    auto run_of = [&](int64_t u) -> Run {
        Run r;
        const int64_t chunk = u / g.n_pos, pos = u - chunk * g.n_pos;
        r.yg = pos / g.nxg; r.xg = pos - r.yg * g.nxg;
        r.plane0 = chunk * g.len;
        r.len = (int)min((int64_t)g.len, g.n_planes - r.plane0);
        r.row0 = r.plane0 * g.S2 + r.yg * kTY * g.S1 + r.xg * kTX;
        return r;
    };

    if (tid >= kConsumers) {
        // ------------------------------------------------ two producer warps ------------------------------------------------
        // Warp kNW feeds the ring, warp kNW + 1 the stages.  A single thread would need ~2,500 cycles for the address arithmetic
        // and the 6-18 bulk copies of one ring slot -- as long as the consumers need for the tile -- so the copies of a slot are
        // issued by one LANE per segment (ring: kTY + 2 lanes, stage: kTY lanes); lane 0 posts the byte count.
        const int lane = tid & 31;
        if (tid < kConsumers + 32) {
            RingPos rp{0u, 1u};                             // next ring load: slot, parity of its "empty" phase (first pass: free)
            const int64_t Ly = g.S2 / g.S1;
            // the tile at (plane, yg, xg) with its halo; planes, lines and in-line positions wrap round the periodic lattice, so
            // the rows on its seams find their neighbours in the slot like everybody else
            auto ring_load = [&](int64_t plane, int64_t yg, int64_t xg) {
                if (lane < kSegs) {
                    mbar_wait(b_rempty + 8 * rp.i, rp.ph);
                    const uint32_t full = b_rfull + 8 * rp.i;
                    if (lane == 0) mbar_expect_tx(full, kSlotBytes);
                    if (plane < 0) plane += g.n_planes;
                    if (plane >= g.n_planes) plane -= g.n_planes;
                    const int64_t x0 = xg * kTX;
                    const bool wrap_lo = x0 == 0, wrap_hi = x0 + kTX == g.S1;
                    int64_t yl = yg * kTY - 1 + lane;
                    if (yl < 0) yl += Ly;
                    if (yl >= Ly) yl -= Ly;
                    const double2 *line = p.x + (plane * g.S2 + yl * g.S1) * kBT;
                    const uint32_t dst = ring0 + rp.i * kSlotBytes + (uint32_t)lane * kSegBytes;
                    const int lo = wrap_lo ? 0 : -1, hi = wrap_hi ? kTX : kTX + 1;       // in-line rows [x0 + lo, x0 + hi) in one piece
                    bulk_g2s(dst + (uint32_t)(lo + 1) * kRowBytes, line + (x0 + lo) * kBT, (uint32_t)(hi - lo) * kRowBytes, full);
                    if (wrap_lo) bulk_g2s(dst, line + (g.S1 - 1) * kBT, kRowBytes, full);
                    if (wrap_hi) bulk_g2s(dst + (uint32_t)(kTX + 1) * kRowBytes, line, kRowBytes, full);
                }
                rp.adv(NR);
            };
            for (int64_t u = blockIdx.x; u < n_runs; u += gridDim.x) {
                const Run r = run_of(u);
                ring_load(r.plane0 - 1, r.yg, r.xg);
                ring_load(r.plane0, r.yg, r.xg);
                for (int j = 0; j < r.len; ++j) ring_load(r.plane0 + j + 1, r.yg, r.xg);
            }
        } else {
            int s = 0;
            uint32_t sph = 1;
            const uint32_t tx = (need_y ? kR * kRowBytes : 0u) + (has_diag ? kR * 8u : 0u);
            for (int64_t u = blockIdx.x; u < n_runs; u += gridDim.x) {
                const Run run = run_of(u);
                for (int j = 0; j < run.len; ++j) {
                    if (lane < kTY) {
                        const int64_t r = run.row0 + (int64_t)j * g.S2 + (int64_t)lane * g.S1;
                        mbar_wait(b_sempty + 8 * s, sph);
                        const uint32_t full = b_sfull + 8 * s;
                        const uint32_t st = stage0 + (uint32_t)s * (uint32_t)g.stage_bytes;
                        if (lane == 0) mbar_expect_tx(full, tx);
                        if (need_y) bulk_g2s(st + g.off_y + lane * (kTX * kRowBytes), p.y + r * kBT, kTX * kRowBytes, full);
                        if (has_diag) bulk_g2s(st + g.off_diag + lane * (kTX * 8), p.diag + r, kTX * 8, full);
                    }
                    if (++s == S) { s = 0; sph ^= 1u; }
                }
            }
        }
        return;
    }

    // ---------------------------------------------------- consumer warps ----------------------------------------------------
    // thread = state `sb` of the tile rows rs and rs + 64 (segments ty0 and ty0 + 2, same in-line position tx)
    const int sb = tid & 7, rs = tid >> 3, ty0 = rs >> 5, tx = rs & 31;
    const uint32_t own0 = (uint32_t)((ty0 + 1) * kSegRows + tx + 1) * kRowBytes + (uint32_t)sb * 16u;   // inside a ring slot
    const uint32_t own1 = own0 + 2u * kSegBytes;
    const uint32_t yo0 = (uint32_t)(ty0 * kTX + tx) * kRowBytes + (uint32_t)sb * 16u, yo1 = yo0 + 2u * kTX * kRowBytes;   // inside the stage's y
    const uint32_t do0 = (uint32_t)(ty0 * kTX + tx) * 8u, do1 = do0 + 2u * kTX * 8u;
    const int64_t roff0 = (int64_t)ty0 * g.S1 + tx, roff1 = roff0 + 2 * g.S1;                             // row - row0 of the tile
    const double t0 = __ldg(p.vtab).x;                      // the one real hopping value
    double s_re = 0.0, s_im = 0.0, s_nn = 0.0;
    const uint32_t off_y = (uint32_t)g.off_y, off_d = (uint32_t)g.off_diag;

    RingPos r0p{0u, 0u}, r1p{1u % NR, 0u}, r2p{2u % NR, 0u};   // the ring loads holding plane z - 1 / z / z + 1 of the tile
    int s = 0;
    uint32_t sph = 0, st = stage0;

    // neighbours of one row from the ring (fast) or entry by entry from global memory (slow); returns their sum
    auto gather_fast = [&](uint32_t bp, uint32_t bo, uint32_t bn, uint32_t own) -> double2 {
        double2 n0, n1, n2, n3, n4, n5;
        lds_c(n0, bp + own);
        lds_c(n1, bo + own - kSegBytes);
        lds_c(n2, bo + own - kRowBytes);
        lds_c(n3, bo + own + kRowBytes);
        lds_c(n4, bo + own + kSegBytes);
        lds_c(n5, bn + own);
        double2 h;
        h.x = ((((n0.x + n1.x) + n2.x) + n3.x) + n4.x) + n5.x;
        h.y = ((((n0.y + n1.y) + n2.y) + n3.y) + n4.y) + n5.y;
        return h;
    };
    auto gather_slow = [&](int64_t row) -> double2 {
        int32_t c[kCH];
#pragma unroll
        for (int j = 0; j < kCH; ++j) c[j] = __ldg(p.ocol + row * kCH + j) & 0x7fffffff;
        double2 n[kCH];
#pragma unroll
        for (int j = 0; j < kCH; ++j) n[j] = ldg_c(p.x + (int64_t)c[j] * kBT + sb);
        double2 h = n[0];
#pragma unroll
        for (int j = 1; j < kCH; ++j) { h.x += n[j].x; h.y += n[j].y; }
        return h;
    };

    // the regular-row bits of a tile's two segments are fetched one tile ahead (an L2 round trip off the critical path)
    uint32_t fwA = 0, fwB = 0;
    if ((int64_t)blockIdx.x < n_runs) {
        const int64_t r0 = run_of(blockIdx.x).row0;
        fwA = __ldg(p.lat_flags + ((r0 + roff0) >> 5)); fwB = __ldg(p.lat_flags + ((r0 + roff1) >> 5));
    }
#pragma unroll 1
    for (int64_t u = blockIdx.x; u < n_runs; u += gridDim.x) {
        const Run run = run_of(u);
        const int len_u = run.len;
        int64_t row0 = run.row0;
        const int64_t next_run_row0 = u + gridDim.x < n_runs ? run_of(u + gridDim.x).row0 : -1;
#pragma unroll 1
        for (int j = 0; j < len_u; ++j, row0 += g.S2) {
            const int64_t rowA = row0 + roff0, rowB = row0 + roff1;
            const int64_t eA = rowA * kBT + sb, eB = rowB * kBT + sb;
            // ---- operands that are not staged (HBM latency: issue first): psi', psi0
            double2 aoldA, aoldB, zA, zB;
            if (NACC > 0) { aoldA = ldg_stream_if(p.acc + eA, need_acc); aoldB = ldg_stream_if(p.acc + eB, need_acc); }
            if (REDUCE) { zA = ldg_stream_if(p.psi0 + eA, true); zB = ldg_stream_if(p.psi0 + eB, true); }
            const bool bitA = (fwA >> (rowA & 31)) & 1u, bitB = (fwB >> (rowB & 31)) & 1u;
            {
                const int64_t nr0 = j + 1 < len_u ? row0 + g.S2 : next_run_row0;
                if (nr0 >= 0) { fwA = __ldg(p.lat_flags + ((nr0 + roff0) >> 5)); fwB = __ldg(p.lat_flags + ((nr0 + roff1) >> 5)); }
            }
            // ---- wait: the ring slots of this tile (the first tile of a run waits for all three), then the stage
            if (j == 0) {
                mbar_wait(b_rfull + 8 * r0p.i, r0p.ph);
                mbar_wait(b_rfull + 8 * r1p.i, r1p.ph);
            }
            mbar_wait(b_rfull + 8 * r2p.i, r2p.ph);
            mbar_wait(b_sfull + 8 * s, sph);
            const uint32_t bp = ring0 + r0p.i * kSlotBytes, bo = ring0 + r1p.i * kSlotBytes, bn = ring0 + r2p.i * kSlotBytes;
            const bool fastA = __all_sync(0xffffffffu, bitA);
            const bool fastB = __all_sync(0xffffffffu, bitB);
            double2 hA, hB;
            if (fastA) hA = gather_fast(bp, bo, bn, own0); else hA = gather_slow(rowA);
            if (fastB) hB = gather_fast(bp, bo, bn, own1); else hB = gather_slow(rowB);
            double2 yA = make_double2(0.0, 0.0), yB = yA, xA = yA, xB = yA;
            double dA = 0.0, dB = 0.0;
            if (need_y) { lds_c(yA, st + off_y + yo0); lds_c(yB, st + off_y + yo1); }
            if (need_xrow) { lds_c(xA, bo + own0); lds_c(xB, bo + own1); }
            if (has_diag) { dA = lds_f64(st + off_d + do0); dB = lds_f64(st + off_d + do1); }
            // Every shared-memory read of this tile must have RETURNED before the stage and the oldest ring slot are handed back to
            // the producers.  A load has returned once an instruction has read its destination register, so the barrier addresses
            // below are made to depend on all of them (`rel` is 0: p.zero is 0, but only at run time).
            const uint32_t rel = (uint32_t)(__double2hiint(hA.x) ^ __double2hiint(hB.x) ^ __double2hiint(yA.x) ^ __double2hiint(yB.x) ^
                                            __double2hiint(xA.x) ^ __double2hiint(xB.x) ^ __double2hiint(dA) ^ __double2hiint(dB)) & (uint32_t)p.zero;
            __syncwarp();
            if ((tid & 31) == 0) {
                mbar_arrive(b_sempty + 8 * s + rel);
                mbar_arrive(b_rempty + 8 * r0p.i + rel);
                if (j == len_u - 1) { mbar_arrive(b_rempty + 8 * r1p.i + rel); mbar_arrive(b_rempty + 8 * r2p.i + rel); }
            }
            if (++s == S) { s = 0; sph ^= 1u; st = stage0; } else st += (uint32_t)g.stage_bytes;
            r0p.adv(NR); r1p.adv(NR); r2p.adv(NR);

            hA.x *= t0; hA.y *= t0; hB.x *= t0; hB.y *= t0;
            if (has_diag) { hA.x = fma(dA, xA.x, hA.x); hA.y = fma(dA, xA.y, hA.y); hB.x = fma(dB, xB.x, hB.x); hB.y = fma(dB, xB.y, hB.y); }
            hA.x *= p.a; hA.y *= p.a; hB.x *= p.a; hB.y *= p.a;
            if (sub_y) { hA.x -= yA.x; hA.y -= yA.y; hB.x -= yB.x; hB.y -= yB.y; }
            if (!REDUCE) { stg_stream(p.y + eA, hA); stg_stream(p.y + eB, hB); }   // T_k: its readers come a whole sweep later
            if (NACC > 0) {
                cfma(aoldA, p.ca, hA); cfma(aoldB, p.ca, hB);
                if (NACC >= 2) { cfma(aoldA, p.cb, xA); cfma(aoldB, p.cb, xB); }
                if (NACC == 3) { cfma(aoldA, p.cc, yA); cfma(aoldB, p.cc, yB); }
                if (REDUCE) {
                    s_re = fma(zA.x, aoldA.x, s_re); s_re = fma(zA.y, aoldA.y, s_re);
                    s_im = fma(zA.x, aoldA.y, s_im); s_im = fma(-zA.y, aoldA.x, s_im);
                    s_nn = fma(aoldA.x, aoldA.x, s_nn); s_nn = fma(aoldA.y, aoldA.y, s_nn);
                    s_re = fma(zB.x, aoldB.x, s_re); s_re = fma(zB.y, aoldB.y, s_re);
                    s_im = fma(zB.x, aoldB.y, s_im); s_im = fma(-zB.y, aoldB.x, s_im);
                    s_nn = fma(aoldB.x, aoldB.x, s_nn); s_nn = fma(aoldB.y, aoldB.y, s_nn);
                    stg(p.acc + eA, aoldA); stg(p.acc + eB, aoldB);          // psi': T_0 of the next step
                } else {
                    stg_stream(p.acc + eA, aoldA); stg_stream(p.acc + eB, aoldB);
                }
            }
        }
        r0p.adv(NR); r0p.adv(NR); r1p.adv(NR); r1p.adv(NR); r2p.adv(NR); r2p.adv(NR);   // a run of len tiles consumes len + 2 ring loads
    }

    if (REDUCE) {
#pragma unroll
        for (int o = 16; o >= 8; o >>= 1) {                 // lanes with equal (lane & 7) hold the same state
            s_re += __shfl_xor_sync(0xffffffffu, s_re, o);
            s_im += __shfl_xor_sync(0xffffffffu, s_im, o);
            s_nn += __shfl_xor_sync(0xffffffffu, s_nn, o);
        }
        const int lane = tid & 31, warp = tid >> 5;
        if (lane < kBT) { red_s[warp][lane][0] = s_re; red_s[warp][lane][1] = s_im; red_s[warp][lane][2] = s_nn; }
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

// Strides and stage layout from the sample row's offsets.  false when they do not describe a lattice this kernel is meant for.
bool make_geom(const TermParams &p, Geom &g)
{
    if (!p.uniform || !p.single_real || p.max_row_off != kCH || p.n_lat_off != kCH || !p.lat_flags || !p.lat_periodic3) return false;
    if (p.n_orb <= 0 || p.n_orb >= ((int64_t)1 << 31)) return false;
    const int64_t S1 = p.lat_delta[4], S2 = p.lat_delta[5];
    if (!(p.lat_delta[0] == -S2 && p.lat_delta[1] == -S1 && p.lat_delta[2] == -1 && p.lat_delta[3] == 1 && S1 > 1 && S2 > S1)) return false;
    if (S1 % kTX != 0 || S2 % (S1 * kTY) != 0 || p.n_orb % S2 != 0 || p.n_orb / S2 < 4) return false;
    if (p.n_regular * 2 < p.n_orb) return false;            // mostly seams: the phased kernel is the better shape
    g.S1 = S1; g.S2 = S2; g.n_planes = p.n_orb / S2;
    g.nxg = (int)(S1 / kTX); g.nyg = (int)(S2 / S1 / kTY);
    g.n_pos = (int64_t)g.nxg * g.nyg;
    g.len = (int)std::min<int64_t>(std::max(1, knob("l3_len", 64)), g.n_planes);
    size_t o = 0;
    g.off_y = (int)o;    o += (size_t)kR * kRowBytes;
    g.off_diag = (int)o; o += (size_t)kR * 8;
    g.stage_bytes = (int)((o + 127) & ~size_t(127));
    g.n_ring = std::min(kMaxRing, std::max(4, knob("l3_ring", 5)));
    g.n_stage = std::min(kMaxStages, std::max(2, knob("l3_stages", 3)));
    return (size_t)g.n_ring * kSlotBytes + (size_t)g.n_stage * g.stage_bytes <= kSmemMax - 4096;
}

template <int NACC, bool REDUCE>
int launch_one(const TermParams &p, const Geom &g, int num_sms, cudaStream_t st, int *grid_out)
{
    const size_t dyn = (size_t)g.n_ring * kSlotBytes + (size_t)g.n_stage * g.stage_bytes;
    auto kern = k_term_l3<NACC, REDUCE>;
    static size_t configured[kMaxDevices] = {0};
    if (p.device < 0 || p.device >= kMaxDevices) return TBPM_EINVAL;
    if (dyn > configured[p.device]) {
        TBPM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kSmemMax - 4096)));
        configured[p.device] = kSmemMax - 4096;
    }
    const int64_t n_runs = g.n_pos * ((g.n_planes + g.len - 1) / g.len);
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>({n_runs, (int64_t)num_sms, (int64_t)kMaxGrid}));
    kern<<<grid, kThreads, dyn, st>>>(p, g);
    count_launches(1);
    *grid_out = grid;
    return TBPM_OK;
}

}  // namespace l3

bool term_l3_supported(int bt, const TermParams &p)
{
    if (bt != l3::kBT || (p.flags & F_SKIP_H) || !knob("l3", 1)) return false;
    const bool red = p.flags & F_REDUCE, wy = p.flags & F_WRITE_Y;
    if (red == wy) return false;
    if (!red && !(p.n_acc == 0 || p.n_acc == 3)) return false;
    if (red && (p.n_acc < 1 || p.n_acc > 3)) return false;
    l3::Geom g;
    return l3::make_geom(p, g);
}

int launch_term_l3(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    l3::Geom g;
    if (!l3::make_geom(p, g)) return TBPM_EINVAL;
    const bool red = p.flags & F_REDUCE;
    if (!red && p.n_acc == 0) return l3::launch_one<0, false>(p, g, num_sms, st, grid_out);
    if (!red && p.n_acc == 3) return l3::launch_one<3, false>(p, g, num_sms, st, grid_out);
    if (red && p.n_acc == 1) return l3::launch_one<1, true>(p, g, num_sms, st, grid_out);
    if (red && p.n_acc == 2) return l3::launch_one<2, true>(p, g, num_sms, st, grid_out);
    if (red && p.n_acc == 3) return l3::launch_one<3, true>(p, g, num_sms, st, grid_out);
    return TBPM_EINVAL;
}

}  // namespace tbpm_detail

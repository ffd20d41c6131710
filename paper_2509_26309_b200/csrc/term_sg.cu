// term_sg.cu -- fused Chebyshev term with the VECTOR rows of a tile staged in shared memory by bulk copies of lattice runs,
// gathered with LDS (tiles of 8 states on uniform lattices: cfg4- and cfg5-like workloads).
//
//   T_k = a*H*T_{k-1} - T_{k-2}  (amxsy) + deferred psi' accumulation + last-term reductions, as term_ph.cuh.
//
// Why (profiles/r1c_l1_line_rate.md): an SM takes one 128-byte line of vector-LOAD traffic every ~2.2 cycles, hit or miss,
// and the fused term asks for 9-12 lines per row of 8 states: 20-26 cycles per row where DRAM needs 15.8.  Shared memory is read
// at 128 B/clk.  On a lattice the j-th neighbours of consecutive rows are consecutive rows (col = row + delta_j away from the
// periodic boundary), so the rows a tile of R rows gathers form a few contiguous SEGMENTS [r0 + lo_s, r0 + hi_s + R) of x -- one
// per group of nearby offsets (cubic: -plane, -line, {-1, 0, +1}, +line, +plane; square with next-nearest neighbours: three).
//   producer warp (one lane): per tile, n_stage tiles ahead, one cp.async.bulk per segment of x, one for y (and psi', psi0 when
//       the term needs them) and one each for the tile's column words / value indices / diagonal: 8-10 copies of 0.5-8 KB;
//   8 consumer warps (thread = row x 2 states): read their column words, and for every entry whose column IS row + delta_j
//       (all but the rows at the periodic boundary) take x from the segment with two conflict-free LDS.128; the others fall
//       back to one LDG.256.  Odd rows read their two 16-byte halves in the opposite order, so a quarter-warp (2 rows x 4
//       lanes) touches all 32 banks once; the halves are put back in order only for the 256-bit stores.
// The offsets delta_j and the segments come from one sample row (build.cu, lat_delta); a matrix that does not follow them
// still gives the right answer through the fallback, only slower.
#include <algorithm>
#include <vector>

#include "term_ph.cuh"

namespace tbpm_detail {
namespace sg {

using namespace ph;

constexpr int kBT = 8, kNW = 8, kConsumers = kNW * 32, kThreads = kConsumers + 32, kR = kConsumers / 4;   // 64 rows per tile
constexpr int kMaxSeg = 8, kMaxSlot = 8, kRowBytes = kBT * 16;

struct Geom {
    int n_seg;
    int seg_lo[kMaxSeg];        // first row of the segment relative to the tile's first row
    int seg_extra[kMaxSeg];     // rows beyond R
    int seg_off[kMaxSeg];       // byte offset inside a stage
    int slot_delta[kMaxSlot];   // expected col - row of entry j
    int slot_addr[kMaxSlot];    // byte offset inside a stage of the row that entry j of the tile's FIRST row gathers
    int centre_addr;            // the same for x[row] itself
    int off_y, off_acc, off_z, off_col, off_idx, off_diag, stage_bytes, n_stage;
};

__device__ __forceinline__ void lds_c(double2 &v, uint32_t a, bool on)     // one complex128 from shared memory, zero when off
{
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %3, 0;\nmov.f64 %0, 0d0000000000000000;\nmov.f64 %1, 0d0000000000000000;\n"
                 "@q ld.shared.v2.f64 {%0, %1}, [%2];\n}"
                 : "=d"(v.x), "=d"(v.y)
                 : "r"(a), "r"((int)on));
}
__device__ __forceinline__ void ldg_pair_if(double2 &lo, double2 &hi, const double2 *p, bool on)   // keeps lo/hi when off
{
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %5, 0;\n@q ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];\n}"
                 : "+d"(lo.x), "+d"(lo.y), "+d"(hi.x), "+d"(hi.y)
                 : "l"(p), "r"((int)on));
}

// CH = entries per row (uniform), VK as in term_ph.cuh (0: table index per entry, 2: one real value).
template <int CH, int VK>
__global__ void __launch_bounds__(kThreads, 1) k_term_sg(const TermParams p, const Geom g)
{
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t bars[2 * kMaxStages];
    __shared__ double red_s[kNW][kBT][3];

    const int tid = threadIdx.x;
    const bool sub_y = p.flags & F_SUB_Y, reduce = p.flags & F_REDUCE, acc_init = p.flags & F_ACC_INIT;
    const int n_acc = p.n_acc;
    const bool need_y = sub_y || n_acc == 3, need_acc = n_acc > 0 && !acc_init, has_diag = p.diag != nullptr;
    const bool need_xrow = n_acc >= 2 || has_diag;
    const int S = g.n_stage;
    const int64_t n_tiles = (p.n_orb + kR - 1) / kR;
    const uint32_t bar0 = smem_u32(bars), smem0 = smem_u32(smem);

    if (tid == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(bar0 + 8 * s, 1); mbar_init(bar0 + 8 * (kMaxStages + s), kNW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (tid >= kConsumers) {
        // ------------------------------------------------ producer warp ------------------------------------------------
        // Every lane issues ONE of the tile's copies (a single thread issuing nine bulk copies per 64-row tile cannot keep up).
        const int lane = tid & 31;
        int s = 0;
        uint32_t ph = 1;
        for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            const int64_t r0 = tile * kR;
            const int rows = (int)min((int64_t)kR, p.n_orb - r0);
            const uint32_t full = bar0 + 8 * s;
            if (lane == 0) mbar_wait(bar0 + 8 * (kMaxStages + s), ph);
            __syncwarp();
            const uint32_t st = smem0 + (uint32_t)s * (uint32_t)g.stage_bytes;
            const uint32_t vb = (uint32_t)rows * kRowBytes;
            uint32_t bytes = 0, dst = 0;
            const void *src = nullptr;
            if (lane < g.n_seg) {                           // the rows of x this tile gathers, one segment per lane
                const int64_t start = r0 + g.seg_lo[lane];
                const int64_t lo = max(start, (int64_t)0), hi = min(start + rows + g.seg_extra[lane], p.n_orb);
                if (hi > lo) { bytes = (uint32_t)(hi - lo) * kRowBytes; dst = st + g.seg_off[lane] + (uint32_t)(lo - start) * kRowBytes; src = p.x + lo * kBT; }
            } else if (lane == 8) {
                if (need_y) { bytes = vb; dst = st + g.off_y; src = p.y + r0 * kBT; }
            } else if (lane == 9) {
                if (need_acc) { bytes = vb; dst = st + g.off_acc; src = p.acc + r0 * kBT; }
            } else if (lane == 10) {
                if (reduce) { bytes = vb; dst = st + g.off_z; src = p.psi0 + r0 * kBT; }
            } else if (lane == 11) {
                bytes = (uint32_t)(((size_t)rows * CH * 4 + 15) & ~size_t(15)); dst = st + g.off_col; src = p.ocol + r0 * CH;
            } else if (lane == 12) {
                if (VK == 0) { bytes = (uint32_t)(((size_t)rows * CH * 2 + 15) & ~size_t(15)); dst = st + g.off_idx; src = p.oidx + r0 * CH; }
            } else if (lane == 13) {
                if (has_diag) { bytes = (uint32_t)((rows * 8 + 15) & ~15); dst = st + g.off_diag; src = p.diag + r0; }
            }
            const uint32_t tx = __reduce_add_sync(0xffffffffu, bytes);
            if (lane == 0) mbar_expect_tx(full, tx);        // before any copy can complete its bytes
            __syncwarp();
            if (bytes) bulk_g2s(dst, src, bytes, full);
            if (++s == S) { s = 0; ph ^= 1u; }
        }
        return;
    }

    // ---------------------------------------------------- consumer warps ----------------------------------------------------
    const int rl = tid >> 2, q = tid & 3, par = rl & 1;     // row of the tile, lane of the row, row parity
    const uint32_t oa = (uint32_t)(2 * q + par) * 16u, ob = (uint32_t)(2 * q + 1 - par) * 16u;   // byte offsets of this thread's two states
    const uint32_t row_off = (uint32_t)rl * kRowBytes;
    double2 t0 = make_double2(0.0, 0.0);
    if (VK == 2) t0 = __ldg(p.vtab);
    double sa_re = 0.0, sa_im = 0.0, sa_nn = 0.0, sb_re = 0.0, sb_im = 0.0, sb_nn = 0.0;

    int s = 0;
    uint32_t ph = 0;
#pragma unroll 1
    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const int64_t row = tile * kR + rl;
        const bool valid = row < p.n_orb;
        const uint32_t st = smem0 + (uint32_t)s * (uint32_t)g.stage_bytes;
        mbar_wait(bar0 + 8 * s, ph);
        // ---- column words (and value indices) of the row
        uint32_t w[CH], id[CH];
        const uint32_t ca = st + g.off_col + (valid ? (uint32_t)rl : 0u) * (CH * 4u);
        const uint32_t ia = st + g.off_idx + (valid ? (uint32_t)rl : 0u) * (CH * 2u);
#pragma unroll
        for (int j = 0; j < CH; j += 2) {
            lds_v2_u32(ca + 4u * j, w[j], w[j + 1]);
            if (VK == 0) { const uint32_t t = lds_u32(ia + 2u * j); id[j] = t & 0xffffu; id[j + 1] = t >> 16; }
            else id[j] = id[j + 1] = 0u;
        }
        // ---- gathers: from the staged segment when the column is where the lattice puts it, else from global memory
        double2 xa[CH], xb[CH];
        bool all_aff = true;
        bool aff[CH];
#pragma unroll
        for (int j = 0; j < CH; ++j) {
            aff[j] = (int64_t)(w[j] & 0x7fffffffu) == row + g.slot_delta[j];
            all_aff = all_aff && (aff[j] || !valid);
        }
        if (__all_sync(0xffffffffu, all_aff)) {
#pragma unroll
            for (int j = 0; j < CH; ++j) {
                const uint32_t a = st + (uint32_t)g.slot_addr[j] + row_off;
                lds_c(xa[j], a + oa, valid);
                lds_c(xb[j], a + ob, valid);
            }
        } else {
#pragma unroll
            for (int j = 0; j < CH; ++j) {
                const uint32_t a = st + (uint32_t)g.slot_addr[j] + row_off;
                lds_c(xa[j], a + oa, valid && aff[j]);
                lds_c(xb[j], a + ob, valid && aff[j]);
                const double2 *src = p.x + (int64_t)(w[j] & 0x7fffffffu) * kBT + 2 * q;
                const bool fb = valid && !aff[j];
                ldg_pair_if(xa[j], xb[j], src, fb && par == 0);      // even rows: a is the first state of the pair
                ldg_pair_if(xb[j], xa[j], src, fb && par == 1);
            }
        }
        // ---- streamed operands of the row, from the stage
        double2 ya, yb, xra, xrb, aa, ab, za, zb;
        lds_c(ya, st + g.off_y + row_off + oa, valid && need_y);
        lds_c(yb, st + g.off_y + row_off + ob, valid && need_y);
        lds_c(xra, st + (uint32_t)g.centre_addr + row_off + oa, valid && need_xrow);
        lds_c(xrb, st + (uint32_t)g.centre_addr + row_off + ob, valid && need_xrow);
        lds_c(aa, st + g.off_acc + row_off + oa, valid && need_acc);
        lds_c(ab, st + g.off_acc + row_off + ob, valid && need_acc);
        lds_c(za, st + g.off_z + row_off + oa, valid && reduce);
        lds_c(zb, st + g.off_z + row_off + ob, valid && reduce);
        const double d = has_diag ? lds_f64(st + g.off_diag + (valid ? (uint32_t)rl : 0u) * 8u) : 0.0;
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(bar0 + 8 * (kMaxStages + s));   // everything this warp needs is in registers
        if (++s == S) { s = 0; ph ^= 1u; }

        // ---- arithmetic
        double2 ha = make_double2(0.0, 0.0), hb = ha;
        if (VK == 2) {
#pragma unroll
            for (int j = 0; j < CH; ++j) { ha.x += xa[j].x; ha.y += xa[j].y; hb.x += xb[j].x; hb.y += xb[j].y; }
            ha.x *= t0.x; ha.y *= t0.x; hb.x *= t0.x; hb.y *= t0.x;
        } else {
            double2 v[CH];
#pragma unroll
            for (int j = 0; j < CH; ++j) v[j] = table_value(ldg_value_if(p.vtab + (id[j] & 0x7fffu), valid), id[j]);
#pragma unroll
            for (int j = 0; j < CH; ++j) { cfma(ha, v[j], xa[j]); cfma(hb, v[j], xb[j]); }
        }
        if (has_diag) { ha.x = fma(d, xra.x, ha.x); ha.y = fma(d, xra.y, ha.y); hb.x = fma(d, xrb.x, hb.x); hb.y = fma(d, xrb.y, hb.y); }
        ha.x *= p.a; ha.y *= p.a; hb.x *= p.a; hb.y *= p.a;
        if (sub_y) { ha.x -= ya.x; ha.y -= ya.y; hb.x -= yb.x; hb.y -= yb.y; }
        if (valid) {
            const int64_t e = row * kBT + 2 * q;
            CVec<2> out;
            if (!reduce) {
                out.v[0] = par ? hb : ha; out.v[1] = par ? ha : hb;
                out.st(p.y + e);
            }
            if (n_acc > 0) {
                cfma(aa, p.ca, ha); cfma(ab, p.ca, hb);
                if (n_acc >= 2) { cfma(aa, p.cb, xra); cfma(ab, p.cb, xrb); }
                if (n_acc == 3) { cfma(aa, p.cc, ya); cfma(ab, p.cc, yb); }
                out.v[0] = par ? ab : aa; out.v[1] = par ? aa : ab;
                if (reduce) {
                    sa_re = fma(za.x, aa.x, sa_re); sa_re = fma(za.y, aa.y, sa_re);
                    sa_im = fma(za.x, aa.y, sa_im); sa_im = fma(-za.y, aa.x, sa_im);
                    sa_nn = fma(aa.x, aa.x, sa_nn); sa_nn = fma(aa.y, aa.y, sa_nn);
                    sb_re = fma(zb.x, ab.x, sb_re); sb_re = fma(zb.y, ab.y, sb_re);
                    sb_im = fma(zb.x, ab.y, sb_im); sb_im = fma(-zb.y, ab.x, sb_im);
                    sb_nn = fma(ab.x, ab.x, sb_nn); sb_nn = fma(ab.y, ab.y, sb_nn);
                    out.st(p.acc + e);
                } else {
                    out.st_stream(p.acc + e);
                }
            }
        }
    }

    if (reduce) {
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
        asm volatile("bar.sync 1, %0;" ::"n"(kConsumers) : "memory");
        if (tid < kBT * 3) {
            const int bb = tid / 3, c = tid % 3;
            double t = 0.0;
#pragma unroll
            for (int w2 = 0; w2 < kNW; ++w2) t += red_s[w2][bb][c];
            p.partial[((int64_t)blockIdx.x * kBT + bb) * 3 + c] = t;
        }
    }
}

// Segments and stage layout from the sample row's offsets (plus offset 0 for x[row]).  Returns false when the offsets do not
// describe a banded lattice this kernel is meant for.
bool make_geom(const TermParams &p, int n_vec_slots, Geom &g)
{
    const int n = p.max_row_off;
    if (n < 2 || n > kMaxSlot || p.n_lat_off != n) return false;
    std::vector<int64_t> d(p.lat_delta, p.lat_delta + n);
    for (int64_t v : d)
        if (v == 0 || v > (int64_t)1 << 28 || v < -((int64_t)1 << 28)) return false;
    std::vector<int64_t> all(d);
    all.push_back(0);
    std::sort(all.begin(), all.end());
    g.n_seg = 0;
    size_t o = 0;
    int64_t lo = all[0], hi = all[0];
    auto close_seg = [&]() -> bool {
        if (g.n_seg == kMaxSeg) return false;
        g.seg_lo[g.n_seg] = (int)lo;
        g.seg_extra[g.n_seg] = (int)(hi - lo);
        g.seg_off[g.n_seg] = (int)o;
        o += (size_t)(kR + (hi - lo)) * kRowBytes;
        ++g.n_seg;
        return true;
    };
    for (size_t i = 1; i < all.size(); ++i) {
        if (all[i] - hi <= 4) hi = all[i];                  // offsets a few rows apart share a segment
        else { if (!close_seg()) return false; lo = hi = all[i]; }
    }
    if (!close_seg()) return false;
    auto addr_of = [&](int64_t delta) {
        for (int k = 0; k < g.n_seg; ++k)
            if (delta >= g.seg_lo[k] && delta <= g.seg_lo[k] + g.seg_extra[k]) return g.seg_off[k] + (int)(delta - g.seg_lo[k]) * kRowBytes;
        return 0;
    };
    for (int j = 0; j < n; ++j) { g.slot_delta[j] = (int)d[j]; g.slot_addr[j] = addr_of(d[j]); }
    g.centre_addr = addr_of(0);
    g.off_y = (int)o;   o += (size_t)kR * kRowBytes;
    g.off_acc = (int)o; o += n_vec_slots >= 2 ? (size_t)kR * kRowBytes : 0;
    g.off_z = (int)o;   o += n_vec_slots >= 3 ? (size_t)kR * kRowBytes : 0;
    g.off_col = (int)o; o += (size_t)kR * n * 4;
    g.off_idx = (int)o; o += (size_t)kR * n * 2;
    o = (o + 15) & ~size_t(15);
    g.off_diag = (int)o; o += (size_t)kR * 8;
    g.stage_bytes = (int)((o + 127) & ~size_t(127));
    return true;
}

template <int CH, int VK>
int launch(const TermParams &p, const Geom &g0, int num_sms, cudaStream_t st, int *grid_out)
{
    Geom g = g0;
    const size_t budget = 220 * 1024;
    g.n_stage = (int)std::min<size_t>(std::min(kMaxStages, std::max(2, env_int("TBPM_STAGES", 6))), budget / g.stage_bytes);
    if (g.n_stage < 2) return TBPM_EINVAL;
    const size_t dyn = (size_t)g.stage_bytes * g.n_stage;
    auto kern = k_term_sg<CH, VK>;
    static size_t configured = 0;
    if (dyn > configured) {
        TBPM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)budget));
        configured = budget;
    }
    const int64_t n_tiles = (p.n_orb + kR - 1) / kR;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>({n_tiles, (int64_t)num_sms, (int64_t)kMaxGrid}));
    kern<<<grid, kThreads, dyn, st>>>(p, g);
    count_launches(1);
    *grid_out = grid;
    return TBPM_OK;
}

}  // namespace sg

bool term_sg_supported(int bt, const TermParams &p)
{
    if (bt != sg::kBT || !p.uniform || p.n_table <= 0 || (p.flags & F_SKIP_H) || !env_int("TBPM_SG", 0)) return false;
    const bool red = p.flags & F_REDUCE, wy = p.flags & F_WRITE_Y;
    if (red == wy) return false;
    const int vk = p.single_real ? 2 : (p.packed ? 1 : 0);
    if (!((vk == 2 && p.max_row_off == 6) || (vk == 0 && p.max_row_off == 8))) return false;
    sg::Geom g;
    return sg::make_geom(p, 3, g) && (size_t)g.stage_bytes * 2 <= 220 * 1024;
}

int launch_term_sg(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    const bool need_acc = p.n_acc > 0 && !(p.flags & F_ACC_INIT), red = p.flags & F_REDUCE;
    sg::Geom g;
    if (!sg::make_geom(p, red ? 3 : (need_acc ? 2 : 1), g)) return TBPM_EINVAL;
    if (p.single_real) return sg::launch<6, 2>(p, g, num_sms, st, grid_out);
    return sg::launch<8, 0>(p, g, num_sms, st, grid_out);
}

}  // namespace tbpm_detail

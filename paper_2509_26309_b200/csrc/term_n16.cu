// term_n16.cu -- fused Chebyshev term for SHORT ROWS with ONE REAL hopping value, tiles of 1, 2 or 4 states (cfg3: honeycomb with
// vacancies, one state; cfg2: honeycomb + Anderson disorder, four states).
//
//   T_k = a*H*T_{k-1} - T_{k-2}  (amxsy)  fused with  psi' += sum c_j T_j  (axpy) and, on the last
//   term of a time step, <psi0|psi'> and <psi'|psi'> (calc_corr_dos) -- the same contract as term_ph.cuh.
//
// Why a kernel of its own (profiles/r2_ncu_cfg3.md): with one state per tile a row is 16 bytes, and the phased kernel spent 258
// instructions per row on it (issue slots 68 % busy, DRAM at 70 %): row offsets, column words, the stage hand-off and 64-bit
// address arithmetic per entry.  Here
//   * the matrix is the builder's `d16` (build.cu, k_near16): W <= 4 slots of 16-bit column offsets per row, slot-major, so a warp
//     reads 64 contiguous bytes per slot -- 2 W bytes per row instead of 4 + 4 n, no row offsets, no shared memory at all (the
//     whole 256 KB of the SM stay L1 for the gathers);
//   * a thread owns one (row, state) element, two tiles in flight: the indices of the tile after next, the loads of the next tile
//     and the arithmetic of this one overlap (software pipeline in registers; 2 x 512 threads per SM);
//   * neighbours at offset +-1 (two of the three on a honeycomb lattice) come from the lane next door by warp shuffle of the
//     tile's own x row, which is read coalesced; only the far neighbour (and the two ends of a warp) is gathered through L1:
//     ~24 instead of ~36 line requests per 32 rows.
// Blocks walk the tiles in linear order, all of them inside one moving window of the vectors (L2 locality), every other term from
// the end (TermParams::reverse), as term_ph.cuh does.
#include <algorithm>

#include "ptx_helpers.cuh"
#include "term.h"

namespace tbpm_detail {
namespace n16 {

// Threads per block, two blocks per SM: the plain term fits 64 registers per thread; the terms that also carry psi' (and psi0) take 80.
__host__ __device__ constexpr int threads_of(int nacc) { return nacc == 0 ? 512 : 384; }

__device__ __forceinline__ double2 ld_gather_if(const double2 *p, bool on)     // read-only path, cacheable; zero when off
{
    double2 v;
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %3, 0;\nmov.f64 %0, 0d0000000000000000;\nmov.f64 %1, 0d0000000000000000;\n"
                 "@q ld.global.nc.v2.f64 {%0, %1}, [%2];\n}"
                 : "=d"(v.x), "=d"(v.y)
                 : "l"(p), "r"((int)on));
    return v;
}
__device__ __forceinline__ double2 ld_stream_if(const double2 *p, bool on)     // read once: evict first
{
    double2 v;
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %3, 0;\nmov.f64 %0, 0d0000000000000000;\nmov.f64 %1, 0d0000000000000000;\n"
                 "@q ld.global.cs.v2.f64 {%0, %1}, [%2];\n}"
                 : "=d"(v.x), "=d"(v.y)
                 : "l"(p), "r"((int)on)
                 : "memory");
    return v;
}
__device__ __forceinline__ double ld_f64_if(const double *p, bool on)
{
    double v;
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %2, 0;\nmov.f64 %0, 0d0000000000000000;\n@q ld.global.nc.f64 %0, [%1];\n}"
                 : "=d"(v)
                 : "l"(p), "r"((int)on));
    return v;
}
__device__ __forceinline__ int ld_s16_if(const int16_t *p, bool on)
{
    int v;
    asm volatile("{\n.reg .pred q;\n.reg .s16 h;\nsetp.ne.b32 q, %2, 0;\nmov.s16 h, 0;\n@q ld.global.nc.s16 h, [%1];\ncvt.s32.s16 %0, h;\n}"
                 : "=r"(v)
                 : "l"(p), "r"((int)on));
    return v;
}
__device__ __forceinline__ void st_f2(double2 *p, double2 v)
{
    asm volatile("st.global.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ void st_f2_stream(double2 *p, double2 v)
{
    asm volatile("st.global.cs.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ double2 shfl_down2(double2 v, int d)
{
    return make_double2(__shfl_down_sync(0xffffffffu, v.x, d), __shfl_down_sync(0xffffffffu, v.y, d));
}
__device__ __forceinline__ double2 shfl_up2(double2 v, int d)
{
    return make_double2(__shfl_up_sync(0xffffffffu, v.x, d), __shfl_up_sync(0xffffffffu, v.y, d));
}

// The loads of one (row, state) element of one tile.
template <int W, int NACC, bool REDUCE> struct Slot {
    int how;              // bit 0: one entry is row + 1 and the lane above holds it; bit 1: row - 1, the lane below
    double d;             // diagonal entry
    double2 y, x, a, z, g[W];
};

template <int BT, int W, int NACC, bool REDUCE, bool DIAG>
__global__ void __launch_bounds__(threads_of(NACC), 2) k_term_n16(const TermParams p)
{
    constexpr int kThreads = threads_of(NACC);
    constexpr int R = kThreads / BT;                        // rows per tile
    __shared__ double red_s[REDUCE ? kThreads / 32 : 1][REDUCE ? BT : 1][3];
    const int tid = threadIdx.x, lane = tid & 31;
    const uint32_t rl = tid / BT, b = tid % BT;
    const bool sub_y = p.flags & F_SUB_Y;
    const bool need_y = sub_y || NACC == 3;
    const bool need_acc = NACC > 0 && !(p.flags & F_ACC_INIT);
    const bool st_ef = p.pol & 1;
    // Rows are 32-bit (n_orb < 2^31, tbpm_build_bytes).  This block's tiles: blockIdx.x, blockIdx.x + gridDim.x, ... -- or the same
    // counted from the last tile (reverse sweep); `row` is this thread's row of the tile being consumed, `drow` the step to the next.
    const uint32_t N = (uint32_t)p.n_orb;
    const uint32_t n_tiles = (N + R - 1) / R;
    const int n_my = blockIdx.x < n_tiles ? (int)((n_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x) : 0;
    const uint32_t drow = p.reverse ? 0u - gridDim.x * (uint32_t)R : gridDim.x * (uint32_t)R;
    uint32_t row = (p.reverse ? n_tiles - 1 - blockIdx.x : blockIdx.x) * (uint32_t)R + rl;
    const double t0 = __ldg(&p.vtab[0].x);
    const bool lane_up = lane + BT < 32, lane_dn = lane >= BT;

    // column offsets of row r (clamped into the matrix: the threads past its end redo the last row and store nothing)
    auto load_idx = [&](uint32_t r, int (&dn)[W]) {
        const uint32_t rc = min(r, N - 1);
        const int16_t *q = p.d16 + (size_t)(rc >> 5) * (W * 32) + (rc & 31u);
#pragma unroll
        for (int j = 0; j < W; ++j) dn[j] = __ldg(q + j * 32);
    };
    // every load of the element: streamed operands, the tile's own x row, and the gathers that no neighbouring lane can serve
    auto issue = [&](Slot<W, NACC, REDUCE> &s, uint32_t r, const int (&dn)[W]) {
        const uint32_t rc = min(r, N - 1);
        const size_t e = (size_t)rc * BT + b;
        s.y = make_double2(0.0, 0.0);
        if (need_y) s.y = __ldcs(p.y + e);
        s.x = __ldg(p.x + e);
        if (NACC > 0) { s.a = make_double2(0.0, 0.0); if (need_acc) s.a = __ldcs(p.acc + e); }
        if (REDUCE) s.z = __ldcs(p.psi0 + e);
        if (DIAG) s.d = __ldg(p.diag + rc);
        s.how = 0;
#pragma unroll
        for (int j = 0; j < W; ++j) {
            const int dj = dn[j];
            const bool up = dj == 1 && lane_up && rc + 1 < N, dw = dj == -1 && lane_dn;
            s.how |= (up ? 1 : 0) | (dw ? 2 : 0);           // at most one entry of a row sits at + 1, at most one at - 1
            uint32_t c = rc + (uint32_t)dj;                 // offsets are stored modulo n_orb (periodic boundaries)
            if (c >= N) c += dj < 0 ? N : 0u - N;
            s.g[j] = ld_gather_if(p.x + (size_t)c * BT + b, dj != 0 && !up && !dw);
        }
    };

    double s_re = 0.0, s_im = 0.0, s_nn = 0.0;
    auto consume = [&](Slot<W, NACC, REDUCE> &s, uint32_t r) {
        const double2 xu = shfl_down2(s.x, BT), xd = shfl_up2(s.x, BT);    // x of row + 1 / row - 1, same state
        double2 h = s.g[0];
#pragma unroll
        for (int j = 1; j < W; ++j) { h.x += s.g[j].x; h.y += s.g[j].y; }
        if (s.how & 1) { h.x += xu.x; h.y += xu.y; }
        if (s.how & 2) { h.x += xd.x; h.y += xd.y; }
        h.x *= t0;
        h.y *= t0;
        if (DIAG) { h.x = fma(s.d, s.x.x, h.x); h.y = fma(s.d, s.x.y, h.y); }
        h.x *= p.a;
        h.y *= p.a;
        if (sub_y) { h.x -= s.y.x; h.y -= s.y.y; }
        if (r < N) {
            const size_t e = (size_t)r * BT + b;
            if (!REDUCE) { if (st_ef) st_f2_stream(p.y + e, h); else st_f2(p.y + e, h); }   // T_k
            if (NACC > 0) {
                double2 a = s.a;
                cfma(a, p.ca, h);
                if (NACC >= 2) cfma(a, p.cb, s.x);
                if (NACC == 3) cfma(a, p.cc, s.y);
                if (REDUCE) {
                    s_re = fma(s.z.x, a.x, s_re);           // conj(z) * psi'
                    s_re = fma(s.z.y, a.y, s_re);
                    s_im = fma(s.z.x, a.y, s_im);
                    s_im = fma(-s.z.y, a.x, s_im);
                    s_nn = fma(a.x, a.x, s_nn);
                    s_nn = fma(a.y, a.y, s_nn);
                    st_f2(p.acc + e, a);                    // psi': T_0 of the next step, gathered right away
                } else {
                    st_f2_stream(p.acc + e, a);
                }
            }
        }
    };

    // Software pipeline over this block's tiles: indices two tiles ahead, loads one tile ahead.
    Slot<W, NACC, REDUCE> A, B;
    int dn[W];
    if (n_my > 0) {
        load_idx(row, dn);
        issue(A, row, dn);
        if (n_my > 1) load_idx(row + drow, dn);
    }
#pragma unroll 1
    for (int i = 0; i < n_my; i += 2) {
        if (i + 1 < n_my) {
            issue(B, row + drow, dn);
            if (i + 2 < n_my) load_idx(row + 2 * drow, dn);
        }
        consume(A, row);
        if (i + 1 >= n_my) break;
        if (i + 2 < n_my) {
            issue(A, row + 2 * drow, dn);
            if (i + 3 < n_my) load_idx(row + 3 * drow, dn);
        }
        consume(B, row + drow);
        row += 2 * drow;
    }

    if (REDUCE) {
#pragma unroll
        for (int o = 16; o >= BT; o >>= 1) {                // lanes with equal (lane % BT) hold the same state
            s_re += __shfl_xor_sync(0xffffffffu, s_re, o);
            s_im += __shfl_xor_sync(0xffffffffu, s_im, o);
            s_nn += __shfl_xor_sync(0xffffffffu, s_nn, o);
        }
        const int warp = tid >> 5;
        if (lane < BT) { red_s[warp][lane][0] = s_re; red_s[warp][lane][1] = s_im; red_s[warp][lane][2] = s_nn; }
        __syncthreads();
        if (tid < BT * 3) {
            const int bb = tid / 3, c = tid % 3;
            double sum = 0.0;
#pragma unroll
            for (int w = 0; w < kThreads / 32; ++w) sum += red_s[w][bb][c];
            p.partial[((int64_t)blockIdx.x * BT + bb) * 3 + c] = sum;
        }
    }
}

template <int BT, int W, int NACC, bool REDUCE>
int launch_one(TermParams p, int num_sms, cudaStream_t st, int *grid_out)
{
    constexpr int kThreads = threads_of(NACC);
    constexpr int R = kThreads / BT;
    p.pol = knob("pol", 1);
    const int64_t need = (p.n_orb + R - 1) / R;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>({need, (int64_t)num_sms * 2, (int64_t)kMaxGrid}));
    if (p.diag) k_term_n16<BT, W, NACC, REDUCE, true><<<grid, kThreads, 0, st>>>(p);
    else k_term_n16<BT, W, NACC, REDUCE, false><<<grid, kThreads, 0, st>>>(p);
    count_launches(1);
    *grid_out = grid;
    return TBPM_OK;
}

template <int BT, int W>
int launch_variant(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    const bool red = p.flags & F_REDUCE;
    if (!red && p.n_acc == 0) return launch_one<BT, W, 0, false>(p, num_sms, st, grid_out);
    if (!red && p.n_acc == 3) return launch_one<BT, W, 3, false>(p, num_sms, st, grid_out);
    if (red && p.n_acc == 1) return launch_one<BT, W, 1, true>(p, num_sms, st, grid_out);
    if (red && p.n_acc == 2) return launch_one<BT, W, 2, true>(p, num_sms, st, grid_out);
    if (red && p.n_acc == 3) return launch_one<BT, W, 3, true>(p, num_sms, st, grid_out);
    return TBPM_EINVAL;
}

template <int BT>
int launch_bt(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    if (p.n16_w == 3) return launch_variant<BT, 3>(p, num_sms, st, grid_out);
    if (p.n16_w == 4) return launch_variant<BT, 4>(p, num_sms, st, grid_out);
    return TBPM_EINVAL;
}

}  // namespace n16

// The builder kept 16-bit column offsets (rows of <= 4 entries within 32767 rows of their own, one real hopping value), the tile
// holds 1, 2 or 4 states, and the term is one of the five (n_acc, reduce) shapes of a time step.
bool term_n16_supported(int bt, const TermParams &p)
{
    if (!p.d16 || (p.n16_w != 3 && p.n16_w != 4) || !p.single_real || p.n_table != 1 || (p.flags & F_SKIP_H)) return false;
    if (bt != 1) return false;                              // wider tiles: the phased kernel's two states per thread are faster
    const bool red = p.flags & F_REDUCE, wy = p.flags & F_WRITE_Y;
    if (red == wy) return false;
    if (!red && !(p.n_acc == 0 || p.n_acc == 3)) return false;
    if (red && (p.n_acc < 1 || p.n_acc > 3)) return false;
    return p.n_orb >= 1;
}

int launch_term_n16(int bt, const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    switch (bt) {
    case 1: return n16::launch_bt<1>(p, num_sms, st, grid_out);
    case 2: return n16::launch_bt<2>(p, num_sms, st, grid_out);
    case 4: return n16::launch_bt<4>(p, num_sms, st, grid_out);
    }
    return TBPM_EINVAL;
}

}  // namespace tbpm_detail

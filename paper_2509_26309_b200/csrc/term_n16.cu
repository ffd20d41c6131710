// term_n16.cu -- fused Chebyshev term for SHORT ROWS with ONE REAL hopping value, tiles of one state (cfg3: honeycomb with vacancies;
// the template also covers tiles of 2 and 4 states with two states per thread, where the phased kernel is as fast and stays in use).
//
//   T_k = a*H*T_{k-1} - T_{k-2}  (amxsy)  fused with  psi' += sum c_j T_j  (axpy) and, on the last
//   term of a time step, <psi0|psi'> and <psi'|psi'> (calc_corr_dos) -- the same contract as term_ph.cuh.
//
// Why a kernel of its own (profiles/r2_ncu_cfg3.md): with one state per tile a row is 16 bytes, and the phased kernel spent 258
// instructions per row on it (issue slots 68 % busy, DRAM at 70 %): row offsets, column words, the stage hand-off and 64-bit
// address arithmetic per entry.  Here
//   * the matrix is the builder's `d16` (build.cu, k_near16): per row one 16-bit FLAG word (has a neighbour at row + 1 / row - 1) and
//     WF <= 4 FAR column offsets, word-major within groups of 32 rows, so a warp reads 64 contiguous bytes per word -- 2 (1 + WF)
//     bytes per row instead of 4 + 4 n, no row offsets, no shared memory at all (the whole 256 KB of the SM stay L1 for the gathers);
//   * a thread owns one (row, state) element, two tiles in flight: the words of the tile after next, the loads of the next tile
//     and the arithmetic of this one overlap (software pipeline in registers; 2 x 512 threads per SM, 32-bit row arithmetic);
//   * the neighbours at row +- 1 (two of the three on a honeycomb lattice) come from the lane next door by warp shuffle of the
//     tile's own x row, which is read coalesced; only the far neighbours -- and, by ONE predicated load, the neighbour beyond either
//     end of a warp -- are gathered through L1.  104 instructions per row; the plain term runs at the DRAM bandwidth (6.3 TB/s).
// Blocks walk the tiles in linear order, all of them inside one moving window of the vectors (L2 locality), every other term from
// the end (TermParams::reverse), as term_ph.cuh does.  An L2 prefetch of the streamed rows some tiles ahead made it slower (342 ->
// 357 -> 434 us per launch at distances 0, 2, 16) and is not part of the kernel.
#include <algorithm>

#include "ptx_helpers.cuh"
#include "term.h"

namespace tbpm_detail {
namespace n16 {

// Threads per block, two blocks per SM: the plain term fits 64 registers per thread; the terms that also carry psi' (and psi0) take 80,
// two states per thread 128.
__host__ __device__ constexpr int threads_of(int nacc, int spt) { return spt == 2 ? 256 : nacc == 0 ? 512 : 384; }

// SPT consecutive complex128 values of one row (SPT = 2: one 256-bit access)
template <int SPT> struct CV;
template <> struct CV<1> {
    double2 v[1];
    __device__ __forceinline__ void zero() { v[0] = make_double2(0.0, 0.0); }
    __device__ __forceinline__ void ld(const double2 *p) { v[0] = __ldg(p); }
    __device__ __forceinline__ void ld_if(const double2 *p, bool on)          // zero when off
    {
        asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %3, 0;\nmov.f64 %0, 0d0000000000000000;\nmov.f64 %1, 0d0000000000000000;\n"
                     "@q ld.global.nc.v2.f64 {%0, %1}, [%2];\n}"
                     : "=d"(v[0].x), "=d"(v[0].y)
                     : "l"(p), "r"((int)on));
    }
    __device__ __forceinline__ void ld_stream(const double2 *p) { v[0] = __ldcs(p); }
    __device__ __forceinline__ void st(double2 *p) const { asm volatile("st.global.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(v[0].x), "d"(v[0].y) : "memory"); }
    __device__ __forceinline__ void st_stream(double2 *p) const
    {
        asm volatile("st.global.cs.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(v[0].x), "d"(v[0].y) : "memory");
    }
};
template <> struct CV<2> {
    double2 v[2];
    __device__ __forceinline__ void zero() { v[0] = v[1] = make_double2(0.0, 0.0); }
    __device__ __forceinline__ void ld(const double2 *p)
    {
        asm volatile("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(v[0].x), "=d"(v[0].y), "=d"(v[1].x), "=d"(v[1].y) : "l"(p));
    }
    __device__ __forceinline__ void ld_if(const double2 *p, bool on)
    {
        asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %5, 0;\nmov.f64 %0, 0d0000000000000000;\nmov.f64 %1, 0d0000000000000000;\n"
                     "mov.f64 %2, 0d0000000000000000;\nmov.f64 %3, 0d0000000000000000;\n"
                     "@q ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];\n}"
                     : "=d"(v[0].x), "=d"(v[0].y), "=d"(v[1].x), "=d"(v[1].y)
                     : "l"(p), "r"((int)on));
    }
    __device__ __forceinline__ void ld_stream(const double2 *p)
    {
        asm volatile("ld.global.L1::no_allocate.L2::evict_first.v4.f64 {%0, %1, %2, %3}, [%4];"
                     : "=d"(v[0].x), "=d"(v[0].y), "=d"(v[1].x), "=d"(v[1].y)
                     : "l"(p)
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

// The loads of one (row, SPT states) element of one tile.
template <int SPT, int WF, int NACC, bool REDUCE> struct Slot {
    int f;                // the row's flag word: bit 0 = it has an entry at row + 1, bit 1 = at row - 1
    double d;             // diagonal entry
    CV<SPT> y, x, a, z, ge, g[WF];
};

// BT states per row, SPT per thread, WF far slots per row.
template <int BT, int SPT, int WF, int NACC, bool REDUCE, bool DIAG>
__global__ void __launch_bounds__(threads_of(NACC, SPT), 2) k_term_n16(const TermParams p)
{
    constexpr int kThreads = threads_of(NACC, SPT);
    constexpr int LPR = BT / SPT;                           // lanes per row
    constexpr int R = kThreads / LPR;                       // rows per tile
    constexpr int S = 1 + WF;                               // 16-bit words per row: flags + far offsets
    __shared__ double red_s[REDUCE ? kThreads / 32 : 1][REDUCE ? BT : 1][3];
    const int tid = threadIdx.x, lane = tid & 31;
    const uint32_t rl = tid / LPR, b = (tid % LPR) * SPT;
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
    // The lane LPR above holds row + 1, the lane LPR below row - 1; the rows at the two ends of a warp gather that neighbour instead
    // (one lane group each, one line request): a lane is at one end at most, so ONE predicated load serves both cases.
    const bool lane_up = lane + LPR < 32, lane_dn = lane >= LPR;
    const int edge_bit = !lane_up ? 1 : !lane_dn ? 2 : 0;
    const int shfl_bits = (lane_up ? 1 : 0) | (lane_dn ? 2 : 0);
    const int edge_off = !lane_up ? BT : -BT;               // in elements

    // flag word and far offsets of row r (clamped into the matrix: the threads past its end redo the last row and store nothing)
    auto load_idx = [&](uint32_t r, int (&dn)[S]) {
        const uint32_t rc = min(r, N - 1);
        const int16_t *q = p.d16 + (size_t)(rc >> 5) * (S * 32) + (rc & 31u);
#pragma unroll
        for (int j = 0; j < S; ++j) dn[j] = __ldg(q + j * 32);
    };
    // every load of the element: streamed operands, the tile's own x row, the far gathers and the edge gather
    auto issue = [&](Slot<SPT, WF, NACC, REDUCE> &s, uint32_t r, const int (&dn)[S]) {
        const uint32_t rc = min(r, N - 1);
        const size_t e = (size_t)rc * BT + b;
        s.y.zero();
        if (need_y) s.y.ld_stream(p.y + e);
        s.x.ld(p.x + e);
        if (NACC > 0) { s.a.zero(); if (need_acc) s.a.ld_stream(p.acc + e); }
        if (REDUCE) s.z.ld_stream(p.psi0 + e);
        if (DIAG) s.d = __ldg(p.diag + rc);
        s.f = dn[0];
        s.ge.ld_if(p.x + e + edge_off, (dn[0] & edge_bit) != 0);
#pragma unroll
        for (int j = 0; j < WF; ++j) {
            const int dj = dn[1 + j];
            uint32_t c = rc + (uint32_t)dj;                 // far offsets are stored modulo n_orb (periodic boundaries)
            if (c >= N) c += dj < 0 ? N : 0u - N;
            s.g[j].ld_if(p.x + (size_t)c * BT + b, dj != 0);
        }
    };

    double s_re[SPT], s_im[SPT], s_nn[SPT];
#pragma unroll
    for (int k = 0; k < SPT; ++k) s_re[k] = s_im[k] = s_nn[k] = 0.0;
    auto consume = [&](Slot<SPT, WF, NACC, REDUCE> &s, uint32_t r) {
        const int use = s.f & shfl_bits;
        CV<SPT> h = s.ge;
#pragma unroll
        for (int k = 0; k < SPT; ++k) {
            const double ux = __shfl_down_sync(0xffffffffu, s.x.v[k].x, LPR), uy = __shfl_down_sync(0xffffffffu, s.x.v[k].y, LPR);
            const double dx = __shfl_up_sync(0xffffffffu, s.x.v[k].x, LPR), dy = __shfl_up_sync(0xffffffffu, s.x.v[k].y, LPR);
#pragma unroll
            for (int j = 0; j < WF; ++j) { h.v[k].x += s.g[j].v[k].x; h.v[k].y += s.g[j].v[k].y; }
            if (use & 1) { h.v[k].x += ux; h.v[k].y += uy; }
            if (use & 2) { h.v[k].x += dx; h.v[k].y += dy; }
            h.v[k].x *= t0;
            h.v[k].y *= t0;
            if (DIAG) { h.v[k].x = fma(s.d, s.x.v[k].x, h.v[k].x); h.v[k].y = fma(s.d, s.x.v[k].y, h.v[k].y); }
            h.v[k].x *= p.a;
            h.v[k].y *= p.a;
            if (sub_y) { h.v[k].x -= s.y.v[k].x; h.v[k].y -= s.y.v[k].y; }
        }
        if (r < N) {
            const size_t e = (size_t)r * BT + b;
            if (!REDUCE) { if (st_ef) h.st_stream(p.y + e); else h.st(p.y + e); }   // T_k
            if (NACC > 0) {
                CV<SPT> a = s.a;
#pragma unroll
                for (int k = 0; k < SPT; ++k) {
                    cfma(a.v[k], p.ca, h.v[k]);
                    if (NACC >= 2) cfma(a.v[k], p.cb, s.x.v[k]);
                    if (NACC == 3) cfma(a.v[k], p.cc, s.y.v[k]);
                    if (REDUCE) {
                        s_re[k] = fma(s.z.v[k].x, a.v[k].x, s_re[k]);       // conj(z) * psi'
                        s_re[k] = fma(s.z.v[k].y, a.v[k].y, s_re[k]);
                        s_im[k] = fma(s.z.v[k].x, a.v[k].y, s_im[k]);
                        s_im[k] = fma(-s.z.v[k].y, a.v[k].x, s_im[k]);
                        s_nn[k] = fma(a.v[k].x, a.v[k].x, s_nn[k]);
                        s_nn[k] = fma(a.v[k].y, a.v[k].y, s_nn[k]);
                    }
                }
                if (REDUCE) a.st(p.acc + e);                // psi': T_0 of the next step, gathered right away
                else a.st_stream(p.acc + e);
            }
        }
    };

    // Software pipeline over this block's tiles: indices two tiles ahead, loads one tile ahead.
    Slot<SPT, WF, NACC, REDUCE> A, B;
    int dn[S];
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
        for (int k = 0; k < SPT; ++k) {                     // lanes with equal (lane % LPR) hold the same states
#pragma unroll
            for (int o = 16; o >= LPR; o >>= 1) {
                s_re[k] += __shfl_xor_sync(0xffffffffu, s_re[k], o);
                s_im[k] += __shfl_xor_sync(0xffffffffu, s_im[k], o);
                s_nn[k] += __shfl_xor_sync(0xffffffffu, s_nn[k], o);
            }
        }
        const int warp = tid >> 5;
        if (lane < LPR) {
#pragma unroll
            for (int k = 0; k < SPT; ++k) {
                red_s[warp][lane * SPT + k][0] = s_re[k];
                red_s[warp][lane * SPT + k][1] = s_im[k];
                red_s[warp][lane * SPT + k][2] = s_nn[k];
            }
        }
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

template <int BT, int WF, int NACC, bool REDUCE>
int launch_one(TermParams p, int num_sms, cudaStream_t st, int *grid_out)
{
    constexpr int SPT = BT >= 2 ? 2 : 1;
    constexpr int kThreads = threads_of(NACC, SPT);
    constexpr int R = kThreads / (BT / SPT);
    p.pol = knob("pol", 1);
    const int64_t need = (p.n_orb + R - 1) / R;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>({need, (int64_t)num_sms * 2, (int64_t)kMaxGrid}));
    if (p.diag) k_term_n16<BT, SPT, WF, NACC, REDUCE, true><<<grid, kThreads, 0, st>>>(p);
    else k_term_n16<BT, SPT, WF, NACC, REDUCE, false><<<grid, kThreads, 0, st>>>(p);
    count_launches(1);
    *grid_out = grid;
    return TBPM_OK;
}

template <int BT, int WF>
int launch_variant(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    const bool red = p.flags & F_REDUCE;
    if (!red && p.n_acc == 0) return launch_one<BT, WF, 0, false>(p, num_sms, st, grid_out);
    if (!red && p.n_acc == 3) return launch_one<BT, WF, 3, false>(p, num_sms, st, grid_out);
    if (red && p.n_acc == 1) return launch_one<BT, WF, 1, true>(p, num_sms, st, grid_out);
    if (red && p.n_acc == 2) return launch_one<BT, WF, 2, true>(p, num_sms, st, grid_out);
    if (red && p.n_acc == 3) return launch_one<BT, WF, 3, true>(p, num_sms, st, grid_out);
    return TBPM_EINVAL;
}

template <int BT>
int launch_bt(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    if (p.n16_w == 1) return launch_variant<BT, 1>(p, num_sms, st, grid_out);
    if (p.n16_w == 2) return launch_variant<BT, 2>(p, num_sms, st, grid_out);
    if (p.n16_w == 4) return launch_variant<BT, 4>(p, num_sms, st, grid_out);
    return TBPM_EINVAL;
}

}  // namespace n16

// The builder kept 16-bit column offsets (rows of <= 4 entries within 32767 rows of their own, one real hopping value), the tile
// holds ONE state, and the term is one of the five (n_acc, reduce) shapes of a time step.
bool term_n16_supported(int bt, const TermParams &p)
{
    if (!p.d16 || (p.n16_w != 1 && p.n16_w != 2 && p.n16_w != 4) || !p.single_real || p.n_table != 1 || (p.flags & F_SKIP_H)) return false;
    if (bt != 1) return false;                              // wider tiles: the phased kernel is as fast (cfg2: 88 us against 90)
    const bool red = p.flags & F_REDUCE, wy = p.flags & F_WRITE_Y;
    if (red == wy) return false;
    if (!red && !(p.n_acc == 0 || p.n_acc == 3)) return false;
    if (red && (p.n_acc < 1 || p.n_acc > 3)) return false;
    return p.n_orb >= 1;
}

int launch_term_n16(int bt, const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    if (bt == 1) return n16::launch_bt<1>(p, num_sms, st, grid_out);
    return TBPM_EINVAL;
}

}  // namespace tbpm_detail

// propagate.cu -- steps a2-a8 of the path: Chebyshev time propagation with the per-step correlation fused in.
//
// What one time step computes (section 2.2.1; coefficients PAPER.md:434):
//     T_0 = psi,  T_1 = (1/s) H T_0,  T_k = (2/s) H T_{k-1} - T_{k-2}   [amxsy, in place over T_{k-2}]
//     psi' = sum_{k<K} c_k T_k                                           [axpy with the complex coefficient]
//     corr = <psi0|psi'>,  norm2 = <psi'|psi'>                           [calc_corr_dos, PAPER.md:965-971]
//
// B200 design (differs from the paper's amxsy + axpy pair):
//   * ONE kernel per Chebyshev term does the SpMV, the subtraction, the accumulation into psi' and (last term) the
//     two dot products.  Vectors of a tile of BT states are interleaved [row][state] so that H is read once per row
//     for all BT states (SpMM) and every gather of x[col] is BT*16 contiguous bytes (128-bit loads).
//   * psi' is touched only every third term: at term k the thread already holds T_k (just computed) and T_{k-2}
//     (the y it read) and reads T_{k-1}[row] (an L1/L2 hit: the same line is being gathered by the neighbouring
//     rows), so three terms are added at once.  Vector traffic falls from 5 to 3.67 streams per term.
//   * H is read from the compressed kernel layout built by build.cu (32-bit row offsets, int32 column, 16-bit index
//     into the table of distinct hopping values, real diagonal).
//   * Persistent grid (blocks = SMs x resident blocks), rows handed out grid-strided so that all SMs sweep one moving
//     window of the vectors (L2 locality of the gather); streaming operands use evict-first loads/stores.
//   * Reductions are deterministic: per-thread sums -> warp shuffles -> shared memory -> one partial per block, then a
//     second tiny kernel adds the block partials in a fixed order.  No floating-point atomics anywhere.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <mutex>
#include <vector>

#include "term.h"

using namespace tbpm_detail;

namespace {

constexpr int kThreads = 256;
constexpr size_t kHeaderBytes = 256;
constexpr size_t kPartialBytes = sizeof(double) * 3 * kMaxBT * kMaxGrid;
constexpr size_t kAuxBytes = 64 * 1024;

__device__ __forceinline__ double2 ld_stream(const double2 *p) { return __ldcs(p); }     // read once: evict first
__device__ __forceinline__ void st_stream(double2 *p, double2 v) { __stcs(p, v); }
// ---------------------------------------------------------------------------------------------------------------------
// The fused Chebyshev term.  Thread -> (row, state b): BT consecutive threads share a row.
// Latency structure: the streaming operands of a row (y, psi', psi0, diagonal, x[row]) do not depend on the row
// offsets, so they are issued first; the row offsets of the NEXT grid-stride iteration are prefetched while the current
// row is processed, which leaves a two-deep dependent chain (column/value index -> gather) per row.
// ---------------------------------------------------------------------------------------------------------------------
// Rows first_row, first_row + stride, ... of one term for state b; the three partial sums of the last term are returned in s_*.
// COH: the vectors were written by OTHER thread blocks earlier in the same kernel (k_small_steps): read them through the L2.
template <int BT, bool TABLE, bool COH>
__device__ __forceinline__ void cheb_term_rows(const TermParams &p, int64_t first_row, int64_t stride, int b, double &s_re, double &s_im,
                                               double &s_nn)
{
    const int flags = p.flags;
    const int n_acc = p.n_acc;
    const bool skip_h = flags & F_SKIP_H;
    const bool need_y = (flags & F_SUB_Y) || n_acc == 3;
    const bool need_xrow = skip_h || n_acc >= 2 || (TABLE && p.diag != nullptr);
    const bool need_acc = n_acc > 0 && !(flags & F_ACC_INIT);
    const bool reduce = flags & F_REDUCE;
    auto ldx = [](const double2 *q) -> double2 { return COH ? __ldcg(q) : __ldg(q); };
    int64_t row = first_row;
    int64_t q0 = 0, q1 = 0;                                 // offsets of the current row (prefetched)
    if (row < p.n_orb && !skip_h) {
        if (TABLE) { q0 = __ldg(p.orp + row); q1 = __ldg(p.orp + row + 1); }
        else { q0 = __ldg(p.rowptr + row); q1 = __ldg(p.rowptr + row + 1); }
    }
    for (; row < p.n_orb; row += stride) {
        const int64_t e = row * BT + b;
        // ---- level 0: everything that needs no index
        double2 yold = make_double2(0.0, 0.0), xrow = yold, aold = yold, z = yold;
        double d = 0.0;
        if (need_y) yold = COH ? __ldcg(p.y + e) : ld_stream(p.y + e);
        if (need_acc) aold = COH ? __ldcg(p.acc + e) : ld_stream(p.acc + e);
        if (reduce) z = COH ? __ldcg(p.psi0 + e) : ld_stream(p.psi0 + e);
        if (need_xrow) xrow = ldx(p.x + e);
        if (TABLE && p.diag != nullptr && !skip_h) d = __ldg(p.diag + row);
        const int64_t nrow = row + stride;
        int64_t nq0 = 0, nq1 = 0;
        if (nrow < p.n_orb && !skip_h) {
            if (TABLE) { nq0 = __ldg(p.orp + nrow); nq1 = __ldg(p.orp + nrow + 1); }
            else { nq0 = __ldg(p.rowptr + nrow); nq1 = __ldg(p.rowptr + nrow + 1); }
        }
        // ---- level 1/2: indices, then gathers
        double2 h = make_double2(0.0, 0.0);
        if (!skip_h) {
            for (int64_t q = q0; q < q1; q += 4) {          // batches of up to 4 independent gathers (predicated tail)
                int32_t c0 = 0, c1 = 0, c2 = 0, c3 = 0;
                double2 v0 = make_double2(0.0, 0.0), v1 = v0, v2 = v0, v3 = v0;
                const bool p1 = q + 1 < q1, p2 = q + 2 < q1, p3 = q + 3 < q1;
                if (TABLE) {
                    uint32_t i0 = 0, i1 = 0, i2 = 0, i3 = 0;
                    c0 = __ldg(p.ocol + q) & 0x7fffffff; i0 = __ldg(p.oidx + q);
                    if (p1) { c1 = __ldg(p.ocol + q + 1) & 0x7fffffff; i1 = __ldg(p.oidx + q + 1); }
                    if (p2) { c2 = __ldg(p.ocol + q + 2) & 0x7fffffff; i2 = __ldg(p.oidx + q + 2); }
                    if (p3) { c3 = __ldg(p.ocol + q + 3) & 0x7fffffff; i3 = __ldg(p.oidx + q + 3); }
                    v0 = table_value(__ldg(p.vtab + (i0 & 0x7fffu)), i0);
                    if (p1) v1 = table_value(__ldg(p.vtab + (i1 & 0x7fffu)), i1);
                    if (p2) v2 = table_value(__ldg(p.vtab + (i2 & 0x7fffu)), i2);
                    if (p3) v3 = table_value(__ldg(p.vtab + (i3 & 0x7fffu)), i3);
                } else {
                    c0 = __ldg(p.col + q); v0 = __ldg(p.val + q);
                    if (p1) { c1 = __ldg(p.col + q + 1); v1 = __ldg(p.val + q + 1); }
                    if (p2) { c2 = __ldg(p.col + q + 2); v2 = __ldg(p.val + q + 2); }
                    if (p3) { c3 = __ldg(p.col + q + 3); v3 = __ldg(p.val + q + 3); }
                }
                const double2 x0 = ldx(p.x + (int64_t)c0 * BT + b);
                double2 x1 = make_double2(0.0, 0.0), x2 = x1, x3 = x1;
                if (p1) x1 = ldx(p.x + (int64_t)c1 * BT + b);
                if (p2) x2 = ldx(p.x + (int64_t)c2 * BT + b);
                if (p3) x3 = ldx(p.x + (int64_t)c3 * BT + b);
                cfma(h, v0, x0);
                cfma(h, v1, x1);
                cfma(h, v2, x2);
                cfma(h, v3, x3);
            }
            h.x = fma(d, xrow.x, h.x);                      // real diagonal (kernel layout only; d = 0 otherwise)
            h.y = fma(d, xrow.y, h.y);
            h.x *= p.a;
            h.y *= p.a;
        } else {
            h = xrow;
        }
        if (flags & F_SUB_Y) { h.x -= yold.x; h.y -= yold.y; }
        if (flags & F_WRITE_Y) p.y[e] = h;                  // T_k: gathered by the next term, keep it cacheable
        if (n_acc > 0) {
            double2 s = aold;
            cfma(s, p.ca, h);
            if (n_acc >= 2) cfma(s, p.cb, xrow);
            if (n_acc == 3) cfma(s, p.cc, yold);
            if (reduce) {
                s_re = fma(z.x, s.x, s_re);                 // conj(z) * s
                s_re = fma(z.y, s.y, s_re);
                s_im = fma(z.x, s.y, s_im);
                s_im = fma(-z.y, s.x, s_im);
                s_nn = fma(s.x, s.x, s_nn);
                s_nn = fma(s.y, s.y, s_nn);
                p.acc[e] = s;                               // psi': T_0 of the next step, gathered right away
            } else {
                if (COH) p.acc[e] = s; else st_stream(p.acc + e, s);
            }
        }
        q0 = nq0;
        q1 = nq1;
    }

}

// per-thread sums -> warp shuffles -> shared memory -> one partial per block (fixed order)
template <int BT, int THREADS>
__device__ __forceinline__ void block_partial(double s_re, double s_im, double s_nn, double *partial, int block)
{
    __shared__ double sm[THREADS / 32][kMaxBT][3];
#pragma unroll
    for (int o = 16; o >= BT; o >>= 1) {                    // lanes with equal (lane % BT) hold the same state
        s_re += __shfl_xor_sync(0xffffffffu, s_re, o);
        s_im += __shfl_xor_sync(0xffffffffu, s_im, o);
        s_nn += __shfl_xor_sync(0xffffffffu, s_nn, o);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane < BT) { sm[warp][lane][0] = s_re; sm[warp][lane][1] = s_im; sm[warp][lane][2] = s_nn; }
    __syncthreads();
    if (threadIdx.x < BT * 3) {
        const int bb = threadIdx.x / 3, c = threadIdx.x % 3;
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < THREADS / 32; ++w) t += sm[w][bb][c];
        partial[((int64_t)block * BT + bb) * 3 + c] = t;
    }
    __syncthreads();
}

template <int BT, bool TABLE, int MINB>
__global__ void __launch_bounds__(kThreads, MINB) k_cheb_term(const TermParams p)
{
    constexpr int kRowsPerBlock = kThreads / BT;
    double s_re = 0.0, s_im = 0.0, s_nn = 0.0;
    cheb_term_rows<BT, TABLE, false>(p, (int64_t)blockIdx.x * kRowsPerBlock + threadIdx.x / BT, (int64_t)gridDim.x * kRowsPerBlock,
                                     threadIdx.x % BT, s_re, s_im, s_nn);
    if (p.flags & F_REDUCE) block_partial<BT, kThreads>(s_re, s_im, s_nn, p.partial, blockIdx.x);
}

// ---------------------------------------------------------------------------------------------------------------------
// Small models (cfg1: 8,192 orbitals, one state) are launch-bound on the path above: 21 launches of ~3 us of device work each per
// time step.  k_small_steps runs ALL time steps of a tile in ONE launch of one thread-block cluster (8 blocks x 1024 threads on 8
// SMs) and keeps the four vectors of the tile (three rotating buffers + the bra) in DISTRIBUTED SHARED MEMORY: block c holds
// elements [c E, (c + 1) E) of each vector, a gather of x[col] is a ld.shared::cluster from the block that owns it (mapa), and
// consecutive terms are separated by a hardware cluster barrier with release / acquire semantics.  A thread owns at most two
// (row, state) elements for the whole run and keeps their column words, hopping values and diagonal in registers; block 0 adds the
// 8 block partials of the last term in a fixed order.  The per-term scalars of the three buffer-rotation phases sit in shared memory.
// Kernel layout with a value table, rows of <= 4 off-diagonal entries, <= 16,384 elements per vector; anything else takes the
// launch-per-term path.  psi is written back to its global buffer at the end (tbpm_get_state).
// ---------------------------------------------------------------------------------------------------------------------
constexpr int kSmallThreads = 1024, kSmallCluster = 8, kSmallClusterMax = 16, kSmallMaxK = 28, kSmallCH = 4, kSmallRPT = 2;
struct TermLite {
    int ix, iy, iacc;             // which of the three rotating buffers holds T_{k-1}, T_{k-2} / T_k, psi'
    int n_acc, flags;
    double a; double2 ca, cb, cc;
};
struct SmallParams {
    const TermLite *terms;        // device [3][K]: terms[slot * K + k] for psi in buffer `slot`
    const uint32_t *orp; const int32_t *ocol; const uint16_t *oidx; const double2 *vtab; const double *diag;
    double2 *buf[3];              // global tile buffers: buf[start_slot] holds psi on entry, buf[final slot] psi on exit
    const double2 *bra;
    int64_t n_orb;
    int E;                        // elements of a vector per block (a multiple of the tile width)
    int K, n_step, start_slot, n_valid, state0, packed, uniform, max_row_off;
    double *corr, *norm2, *partial;
};
__device__ __forceinline__ double2 ld_dsmem(uint32_t local_addr, uint32_t rank)
{
    uint32_t ra;
    double2 v;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(local_addr), "r"(rank));
    asm volatile("ld.shared::cluster.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(ra) : "memory");
    return v;
}
template <int BT>
__global__ void __launch_bounds__(kSmallThreads, 1) k_small_steps(const SmallParams sp)
{
    extern __shared__ __align__(16) unsigned char small_smem[];          // [4][E] complex128: buffers 0..2, bra
    __shared__ TermLite tl[3 * kSmallMaxK];
    for (int i = threadIdx.x; i < 3 * sp.K * (int)(sizeof(TermLite) / 4); i += kSmallThreads)
        reinterpret_cast<uint32_t *>(tl)[i] = __ldg(reinterpret_cast<const uint32_t *>(sp.terms) + i);
    double2 *vec = reinterpret_cast<double2 *>(small_smem);
    const uint32_t vec0 = (uint32_t)__cvta_generic_to_shared(vec);
    const int E = sp.E, b = threadIdx.x % BT;
    const int64_t n_el = sp.n_orb * BT, e0 = (int64_t)blockIdx.x * E;
    // the thread's elements (local index le, -1: none) and their matrix rows, for the whole run
    int le[kSmallRPT];
    int32_t col[kSmallRPT][kSmallCH];       // element index (col * BT + b) of each neighbour, split below into (owner, local)
    double2 val[kSmallRPT][kSmallCH];
    double dg[kSmallRPT];
    int nr[kSmallRPT];
#pragma unroll
    for (int i = 0; i < kSmallRPT; ++i) {
        le[i] = (int)threadIdx.x + i * kSmallThreads;
        const int64_t e = e0 + le[i];
        nr[i] = 0; dg[i] = 0.0;
#pragma unroll
        for (int j = 0; j < kSmallCH; ++j) { col[i][j] = 0; val[i][j] = make_double2(0.0, 0.0); }
        if (le[i] >= E || e >= n_el) { le[i] = -1; continue; }
        const int64_t row = e / BT;                         // E is a multiple of BT: e % BT == threadIdx.x % BT == b
        const uint32_t q0 = sp.uniform ? (uint32_t)row * (uint32_t)sp.max_row_off : __ldg(sp.orp + row);
        const uint32_t q1 = sp.uniform ? q0 + (uint32_t)sp.max_row_off : __ldg(sp.orp + row + 1);
        nr[i] = (int)(q1 - q0);
        for (int j = 0; j < nr[i]; ++j) {
            const uint32_t w = (uint32_t)__ldg(sp.ocol + q0 + j);
            const uint32_t id = sp.packed ? (w >> 31) << 15 : (uint32_t)__ldg(sp.oidx + q0 + j);
            col[i][j] = (int32_t)((w & 0x7fffffffu) * BT + b);
            val[i][j] = table_value(__ldg(sp.vtab + (id & 0x7fffu)), id);
        }
        if (sp.diag) dg[i] = __ldg(sp.diag + row);
        // psi and the bra of the tile come in from global memory; the other two buffers are written before they are read
        vec[(size_t)sp.start_slot * E + le[i]] = sp.buf[sp.start_slot][e];
        vec[(size_t)3 * E + le[i]] = sp.bra[e];
    }
    __syncthreads();
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
    int slot = sp.start_slot;
    for (int n = 0; n < sp.n_step; ++n) {
        for (int k = 1; k < sp.K; ++k) {
            const TermLite &t = tl[slot * sp.K + k];
            const bool sub_y = t.flags & F_SUB_Y, reduce = t.flags & F_REDUCE, wy = t.flags & F_WRITE_Y;
            const bool need_y = sub_y || t.n_acc == 3, need_acc = t.n_acc > 0 && !(t.flags & F_ACC_INIT);
            const uint32_t xbase = vec0 + (uint32_t)t.ix * (uint32_t)E * 16u;
            double2 *yv = vec + (size_t)t.iy * E, *av = vec + (size_t)t.iacc * E;
            const double2 *xl = vec + (size_t)t.ix * E, *zv = vec + (size_t)3 * E;
            double s_re = 0.0, s_im = 0.0, s_nn = 0.0;
#pragma unroll
            for (int i = 0; i < kSmallRPT; ++i) {
                if (le[i] < 0) continue;
                double2 xv[kSmallCH];
#pragma unroll
                for (int j = 0; j < kSmallCH; ++j) {
                    xv[j] = make_double2(0.0, 0.0);
                    if (j < nr[i]) { const uint32_t owner = (uint32_t)col[i][j] / (uint32_t)E, loc = (uint32_t)col[i][j] - owner * (uint32_t)E; xv[j] = ld_dsmem(xbase + loc * 16u, owner); }
                }
                const double2 xrow = xl[le[i]];
                double2 yold = make_double2(0.0, 0.0), aold = yold, z = yold;
                if (need_y) yold = yv[le[i]];
                if (need_acc) aold = av[le[i]];
                if (reduce) z = zv[le[i]];
                double2 h = make_double2(0.0, 0.0);
#pragma unroll
                for (int j = 0; j < kSmallCH; ++j) cfma(h, val[i][j], xv[j]);
                h.x = fma(dg[i], xrow.x, h.x); h.y = fma(dg[i], xrow.y, h.y);
                h.x *= t.a; h.y *= t.a;
                if (sub_y) { h.x -= yold.x; h.y -= yold.y; }
                if (wy) yv[le[i]] = h;
                if (t.n_acc > 0) {
                    double2 s = aold;
                    cfma(s, t.ca, h);
                    if (t.n_acc >= 2) cfma(s, t.cb, xrow);
                    if (t.n_acc == 3) cfma(s, t.cc, yold);
                    av[le[i]] = s;
                    if (reduce) {
                        s_re = fma(z.x, s.x, s_re); s_re = fma(z.y, s.y, s_re);
                        s_im = fma(z.x, s.y, s_im); s_im = fma(-z.y, s.x, s_im);
                        s_nn = fma(s.x, s.x, s_nn); s_nn = fma(s.y, s.y, s_nn);
                    }
                }
            }
            if (reduce) block_partial<BT, kSmallThreads>(s_re, s_im, s_nn, sp.partial, blockIdx.x);
            // T_k in shared memory (and the partials in global memory) become visible to the whole cluster
            if (reduce) __threadfence();
            asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
        }
        if (blockIdx.x == 0 && threadIdx.x < sp.n_valid * 3) {
            const int bb = threadIdx.x / 3, c = threadIdx.x % 3;
            double tsum = 0.0;
            for (int g = 0; g < (int)gridDim.x; ++g) tsum += __ldcg(sp.partial + ((int64_t)g * BT + bb) * 3 + c);
            const int64_t at = (int64_t)(sp.state0 + bb) * sp.n_step + n;
            if (c < 2) sp.corr[2 * at + c] = tsum;
            else if (sp.norm2) sp.norm2[at] = tsum;
        }
        slot = (slot + 2) % 3;
    }
#pragma unroll
    for (int i = 0; i < kSmallRPT; ++i)
        if (le[i] >= 0) sp.buf[slot][e0 + le[i]] = vec[(size_t)slot * E + le[i]];
}

// NEXT-4, dynamic polarisation: a DIAGONAL complex operator d (the density operator exp(i q.r)) on one tile of interleaved states.
__global__ void k_diag_apply(const double2 *__restrict__ d, const double2 *__restrict__ x, double2 *y, int64_t n_orb, int bt)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_orb * bt; i += (int64_t)gridDim.x * blockDim.x) {
        const double2 dv = d[i / bt], xv = x[i];
        y[i] = make_double2(dv.x * xv.x - dv.y * xv.y, dv.x * xv.y + dv.y * xv.x);
    }
}
// block partials of <bra| d |x> per state, in the layout k_reduce_final reads ([block][bt][3]; the third component is unused)
template <int BT>
__global__ void __launch_bounds__(256) k_diag_dot(const double2 *__restrict__ d, const double2 *__restrict__ x, const double2 *__restrict__ bra,
                                                  int64_t n_orb, double *partial)
{
    double s_re = 0.0, s_im = 0.0, s_nn = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_orb * BT; i += (int64_t)gridDim.x * blockDim.x) {   // stride % BT == 0
        const double2 dv = d[i / BT], xv = x[i], z = bra[i];
        const double2 w = make_double2(dv.x * xv.x - dv.y * xv.y, dv.x * xv.y + dv.y * xv.x);
        s_re = fma(z.x, w.x, s_re); s_re = fma(z.y, w.y, s_re);
        s_im = fma(z.x, w.y, s_im); s_im = fma(-z.y, w.x, s_im);
    }
    block_partial<BT, 256>(s_re, s_im, s_nn, partial, blockIdx.x);
}

// Sum the block partials in a fixed order: block = state, warp = component, lanes stride over the partials.
__global__ void k_reduce_final(const double *__restrict__ partial, int n_blocks, int bt, int n_valid, int state0, int n_step, int step,
                               double *corr, double *norm2)
{
    const int bb = blockIdx.x, c = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (bb >= n_valid) return;
    double t = 0.0;
    for (int k = lane; k < n_blocks; k += 32) t += partial[((int64_t)k * bt + bb) * 3 + c];
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if (lane == 0) {
        const int64_t at = (int64_t)(state0 + bb) * n_step + step;
        if (c < 2) corr[2 * at + c] = t;
        else if (norm2) norm2[at] = t;
    }
}

// a2: state-major psi0 -> interleaved tile buffers (psi and the bra); states beyond n_valid are zero padding.
__global__ void k_interleave(const double2 *__restrict__ psi0, int64_t n_orb, int state0, int n_valid, int bt, double2 *psi, double2 *bra)
{
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_orb * bt) return;
    const int b = (int)(t % bt);
    const int64_t row = t / bt;
    double2 v = make_double2(0.0, 0.0);
    if (b < n_valid) v = psi0[(int64_t)(state0 + b) * n_orb + row];
    psi[t] = v;
    bra[t] = v;
}

// a8: unit vectors on the given sites
__global__ void k_unit_states(const int64_t *__restrict__ sites, int state0, int n_valid, int bt, double2 *psi, double2 *bra)
{
    int b = threadIdx.x;
    if (b >= n_valid) return;
    const int64_t at = sites[state0 + b] * bt + b;
    psi[at] = make_double2(1.0, 0.0);
    bra[at] = make_double2(1.0, 0.0);
}

// tbpm_get_state: one state of a tile buffer [row][bt] -> caller order
__global__ void k_get_state(const double2 *__restrict__ psi, int64_t n_orb, int bt, int b, double2 *out)
{
    for (int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; row < n_orb; row += (int64_t)gridDim.x * blockDim.x)
        out[row] = psi[row * bt + b];
}


// NEXT-3 (quasi-eigenstates): qe[e][i] (+)= c_e * psi[i] on one tile of interleaved states, for up to kMaxEnergy energies.
constexpr int kMaxEnergy = 16;
struct QeCoef { double2 c[kMaxEnergy]; };
__global__ void k_qe_axpy(const double2 *__restrict__ psi, int64_t n_el, int n_e, QeCoef cf, size_t stride, double2 *qe, int init)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_el; i += (int64_t)gridDim.x * blockDim.x) {
        const double2 v = psi[i];
        for (int e = 0; e < n_e; ++e) {
            double2 *q = qe + (size_t)e * stride + i;
            double2 s = init ? make_double2(0.0, 0.0) : *q;
            cfma(s, cf.c[e], v);
            *q = s;
        }
    }
}
// interleaved tile buffers [e][row][bt] -> caller order qe[state0 + b][e][row]
__global__ void k_qe_export(const double2 *__restrict__ qe_ws, size_t stride, int64_t n_orb, int bt, int n_valid, int state0, int n_e, double2 *out)
{
    const int64_t total = n_orb * n_valid * n_e;
    for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
        const int64_t row = t % n_orb;
        const int e = (int)((t / n_orb) % n_e), b = (int)(t / (n_orb * n_e));
        out[((int64_t)(state0 + b) * n_e + e) * n_orb + row] = qe_ws[(size_t)e * stride + row * bt + b];
    }
}

// NEXT-2 (Haydock recursion), per tile of interleaved states.  Vectors are kept UNNORMALISED (u_n = beta_n phi_n) so that one
// iteration is two sweeps: t = H u_n with <u_n|t> (the fused last-term kernel), then
//     u_{n+1} = t / beta_n - (a_n / beta_n) u_n - (beta_n / beta_{n-1}) u_{n-1},   a_n = Re<u_n|t> / beta_n^2,   b_{n+1} = ||u_{n+1}||
// which is the textbook  b_{n+1} phi_{n+1} = H phi_n - a_n phi_n - b_n phi_{n-1}  with b_n = beta_n.
// sc[b] = {Re<u_n|t>, beta_n, beta_{n-1}, unused}; a zero beta (Krylov space exhausted, or a padding state) gives zeros from then on.
__global__ void k_haydock_update(const double2 *__restrict__ t, const double2 *__restrict__ u, double2 *__restrict__ u_prev, int64_t n_orb, int bt,
                                 const double *__restrict__ sc, double *partial)
{
    __shared__ double sm[256 / 32][kMaxBT];
    const int b = threadIdx.x % bt;
    const double dot = sc[4 * b], beta = sc[4 * b + 1], beta_p = sc[4 * b + 2];
    const double ib = beta > 0.0 ? 1.0 / beta : 0.0;
    const double a_n = dot * ib * ib;
    const double c_prev = beta_p > 0.0 ? beta / beta_p : 0.0;
    double nn = 0.0;
    const int64_t n_el = n_orb * bt;
    // The grid is small (its partials live in the 64 KB aux area), so every thread keeps EIGHT elements in flight: 24 independent
    // 16-byte loads before the first use (~170 KB per SM; with one element per trip the kernel ran at 4.9 TB/s).
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;              // a multiple of bt: a thread stays with its state
    auto one = [&](int64_t i, double2 tv, double2 uv, double2 pv) {
        double2 w;
        w.x = (tv.x - a_n * uv.x) * ib - c_prev * pv.x;
        w.y = (tv.y - a_n * uv.y) * ib - c_prev * pv.y;
        u_prev[i] = w;
        nn = fma(w.x, w.x, nn);
        nn = fma(w.y, w.y, nn);
    };
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + 7 * stride < n_el; i += 8 * stride) {
        double2 tv[8], uv[8], pv[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) { tv[k] = __ldcs(t + i + k * stride); uv[k] = __ldcs(u + i + k * stride); pv[k] = __ldcs(u_prev + i + k * stride); }
#pragma unroll
        for (int k = 0; k < 8; ++k) one(i + k * stride, tv[k], uv[k], pv[k]);
    }
    for (; i < n_el; i += stride) one(i, __ldcs(t + i), __ldcs(u + i), __ldcs(u_prev + i));
    for (int o = 16; o >= bt; o >>= 1) nn += __shfl_xor_sync(0xffffffffu, nn, o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane < bt) sm[warp][lane] = nn;
    __syncthreads();
    if (threadIdx.x < bt) {
        double s = 0.0;
        for (int w2 = 0; w2 < 256 / 32; ++w2) s += sm[w2][threadIdx.x];
        partial[(int64_t)blockIdx.x * bt + threadIdx.x] = s;
    }
}
// block = state: a_n, b_{n+1} out; scalars rotated for the next iteration.  dot_partial: [grid_dot][bt][3] of the term kernel.
__global__ void k_haydock_scalars(const double *__restrict__ dot_partial, int grid_dot, int bt, double *sc, int phase,
                                  const double *__restrict__ nn_partial, int grid_nn, int n_valid, int state0, int n_iter, int it, double *a_out,
                                  double *b_out)
{
    const int b = blockIdx.x, lane = threadIdx.x;
    double s = 0.0;
    if (phase == 0) {                                       // after the H application: Re<u_n|t>
        for (int k = lane; k < grid_dot; k += 32) s += dot_partial[((int64_t)k * bt + b) * 3];
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) sc[4 * b] = s;
    } else {                                                // after the update: beta_{n+1}; publish a_n, b_{n+1}
        for (int k = lane; k < grid_nn; k += 32) s += nn_partial[(int64_t)k * bt + b];
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) {
            const double beta = sc[4 * b + 1], dot = sc[4 * b];
            const double a_n = beta > 0.0 ? dot / (beta * beta) : 0.0, bn = sqrt(s);
            if (b < n_valid) {
                a_out[(int64_t)(state0 + b) * n_iter + it] = a_n;
                b_out[(int64_t)(state0 + b) * n_iter + it] = bn;
            }
            sc[4 * b + 2] = beta;
            sc[4 * b + 1] = bn;
        }
    }
}
__global__ void k_haydock_init(double *sc, int bt, int n_valid)
{
    const int b = threadIdx.x;
    if (b < bt) { sc[4 * b] = 0.0; sc[4 * b + 1] = b < n_valid ? 1.0 : 0.0; sc[4 * b + 2] = 0.0; sc[4 * b + 3] = 0.0; }
}

// ---------------------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------------------
int pow2_ceil(int n)
{
    int p = 1;
    while (p < n) p <<= 1;
    return p;
}

struct Plan {
    int tile;            // states per full tile
    int n_tile;
    int last_bt;         // padded size of the last tile
    size_t full_vec;     // bytes of one vector buffer of a full tile
    size_t sites_off, partial_off, aux_off, vec0_off, total;
};

Plan make_plan(int64_t n_orb, int n_state, int tile_max)
{
    Plan P{};
    P.tile = std::min(tile_max, pow2_ceil(std::max(n_state, 1)));
    P.n_tile = (std::max(n_state, 1) + P.tile - 1) / P.tile;
    const int rest = std::max(n_state, 1) - (P.n_tile - 1) * P.tile;
    P.last_bt = pow2_ceil(rest);
    P.full_vec = align_up((size_t)n_orb * P.tile * sizeof(double2));
    size_t o = kHeaderBytes;
    P.sites_off = o;
    o += align_up(sizeof(int64_t) * (size_t)std::max(n_state, 1));
    P.partial_off = o;
    o += kPartialBytes;
    P.aux_off = o;                                        // scalars and norm partials of tbpm_haydock
    o += kAuxBytes;
    P.vec0_off = o;
    o += (size_t)P.n_tile * 4 * P.full_vec;
    P.total = o;
    return P;
}

template <int BT, bool TABLE>
int launch_term_t(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    static int blocks_per_sm[kMaxDevices] = {0};           // per device
    if (p.device < 0 || p.device >= kMaxDevices) return TBPM_EINVAL;
    if (blocks_per_sm[p.device] == 0) {
        int nb = 0;
        TBPM_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_cheb_term<BT, TABLE, 4>, kThreads, 0));
        blocks_per_sm[p.device] = std::max(nb, 1);
    }
    constexpr int kRowsPerBlock = kThreads / BT;
    const int64_t need = (p.n_orb + kRowsPerBlock - 1) / kRowsPerBlock;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>({need, (int64_t)num_sms * blocks_per_sm[p.device], (int64_t)kMaxGrid}));
    k_cheb_term<BT, TABLE, 4><<<grid, kThreads, 0, st>>>(p);
    count_launches(1);
    *grid_out = grid;
    return TBPM_OK;
}

// One Chebyshev term.  TBPM_OPT_KERNEL = 0: tiles of 8 states on a lattice the builder recognised run on term_l3.cu
// (three-dimensional, one real hopping value), term_sq.cu (square + next-nearest neighbours, in-line hoppings) or term_rw.cu (other
// strides of whole 128-row tiles); the phased kernel (term_ph.cuh) runs whenever it has an instantiation for the term and its
// stages fit (kernel layout with a value table, tiles of 1-8 states, rows of up to a few dozen entries); everything else -- no
// table, tiles of 16 / 32 states, long rows, tau = 0 -- runs on the general kernel k_cheb_term.  1: general kernel only;
// 2: no lattice kernel; 3: of the lattice kernels only term_rw.
int launch_term(int bt, bool table, int kernel_opt, const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    if (kernel_opt == 4) kernel_opt = 0;                  // 4 only switches the two-terms-per-sweep path of run() off
    const bool general_only = kernel_opt == 1;
    if (table && kernel_opt == 0 && term_l3_supported(bt, p)) return launch_term_l3(p, num_sms, st, grid_out);
    if (table && kernel_opt == 0 && term_sq_supported(bt, p)) return launch_term_sq(p, num_sms, st, grid_out);
    if (table && (kernel_opt == 0 || kernel_opt == 3) && term_rw_supported(bt, p)) return launch_term_rw(p, num_sms, st, grid_out);
    if (table && kernel_opt == 0 && term_n16_supported(bt, p)) return launch_term_n16(bt, p, num_sms, st, grid_out);
    if (table && !general_only && term_ph_supported(bt, p)) {
        switch (bt) {
        case 1: return launch_term_ph_bt1(p, num_sms, st, grid_out);
        case 2: return launch_term_ph_bt2(p, num_sms, st, grid_out);
        case 4: return launch_term_ph_bt4(p, num_sms, st, grid_out);
        case 8: return launch_term_ph_bt8(p, num_sms, st, grid_out);
        }
    }
#define TBPM_CASE(B)                                                                     \
    case B:                                                                              \
        return table ? launch_term_t<B, true>(p, num_sms, st, grid_out) : launch_term_t<B, false>(p, num_sms, st, grid_out);
    switch (bt) {
        TBPM_CASE(1)
        TBPM_CASE(2)
        TBPM_CASE(4)
        TBPM_CASE(8)
        TBPM_CASE(16)
        TBPM_CASE(32)
    }
#undef TBPM_CASE
    return TBPM_EINVAL;
}

// Launch parameters of the K - 1 Chebyshev terms of one time step (psi in `psi`, scratch `t1`, psi' built in `acc`).
// T_k overwrites T_{k-2}: T_0 = psi, T_1 -> t1, T_2 -> psi's buffer, ...; psi' is touched on every third term and on
// the last one, which also carries the reduction and does not store T_{K-1} (it is never read again).
void step_terms(const TermParams &base, int K, const std::vector<double> &cf, double rescale, bool reverse_odd, double2 *psi,
                double2 *t1, double2 *acc, std::vector<TermParams> &term)
{
    auto C = [&](int k) { return make_double2(cf[2 * k], cf[2 * k + 1]); };
    term.assign((size_t)K, base);
    int flushed = -1;                                     // highest term already added to psi'
    for (int k = 1; k < K; ++k) {
        TermParams &tp = term[k];
        tp.x = (k % 2 == 1) ? psi : t1;                   // T_{k-1}
        tp.y = (k % 2 == 1) ? t1 : psi;                   // T_{k-2} -> T_k
        tp.acc = acc;
        tp.a = (k == 1 ? 1.0 : 2.0) / rescale;
        int flags = F_WRITE_Y | (k >= 2 ? F_SUB_Y : 0);
        const bool last = (k == K - 1);
        tp.n_acc = 0;
        if (k % 3 == 2 || last) {                         // flush terms flushed+1 .. k (at most 3)
            tp.n_acc = k - flushed;
            tp.ca = C(k);
            tp.cb = tp.n_acc >= 2 ? C(k - 1) : make_double2(0.0, 0.0);
            tp.cc = tp.n_acc == 3 ? C(k - 2) : make_double2(0.0, 0.0);
            if (flushed < 0) flags |= F_ACC_INIT;
            flushed = k;
        }
        if (last) { flags |= F_REDUCE; flags &= ~F_WRITE_Y; }
        tp.flags = flags;
        tp.reverse = reverse_odd ? (k & 1) : 0;
        if (tp.reverse) tp.pf_lead = -tp.pf_lead;
    }
}

// The same time step with TWO terms per launch (term_sq2.cu).  ops[i].pair: launch_pair_sq, else launch_term (only a leading single
// term when K - 1 is odd).  Buffers: psi (T_0), t1, and the two extra vectors e1, e2; a pair reads two of the four and writes the
// other two (T_{k-2} is read with a halo, so nothing is updated in place).  psi' (acc) is touched when the oldest term not yet added
// would otherwise leave the pair's window {k-2 .. k+1}: every second pair, four terms at a time.
struct StepOp { bool pair; TermParams tp; };
void step_pairs(const TermParams &base, int K, const std::vector<double> &cf, double rescale, double2 *psi, double2 *t1, double2 *acc,
                double2 *e1, double2 *e2, std::vector<StepOp> &ops)
{
    auto C = [&](int k) { return make_double2(cf[2 * k], cf[2 * k + 1]); };
    const double2 zero = make_double2(0.0, 0.0);
    ops.clear();
    int oldest = 0;                                       // lowest term not yet added to psi' (terms oldest .. k - 1 are pending)
    bool any_flush = false;
    double2 *X = psi, *Y = t1, *F1 = e1, *F2 = e2;        // T_{k-1}, T_{k-2}, and the two buffers free to be written
    int k = 1;
    if ((K - 1) % 2 == 1) {                               // odd number of terms: T_1 on its own, in t1
        StepOp op{false, base};
        op.tp.x = psi; op.tp.y = t1; op.tp.acc = acc; op.tp.a = 1.0 / rescale; op.tp.n_acc = 0; op.tp.flags = F_WRITE_Y; op.tp.reverse = 0;
        ops.push_back(op);
        X = t1; Y = psi;
        k = 2;
    }
    for (; k + 1 < K; k += 2) {
        StepOp op{true, base};
        TermParams &tp = op.tp;
        tp.x = X; tp.y = Y; tp.out1 = F1; tp.out2 = F2; tp.acc = acc;
        tp.a = (k == 1 ? 1.0 : 2.0) / rescale;
        tp.a2 = 2.0 / rescale;
        int flags = k >= 2 ? F_SUB_Y : 0;
        const bool last = k + 1 == K - 1;
        tp.n_acc = 0;
        tp.ca = tp.cb = tp.cc = tp.cd = zero;
        if (oldest < k || last) {                         // terms oldest .. k + 1, all inside the window (oldest >= k - 2)
            tp.n_acc = k + 2 - oldest;
            tp.ca = C(k + 1); tp.cb = C(k);
            if (oldest <= k - 1) tp.cc = C(k - 1);
            if (oldest <= k - 2) tp.cd = C(k - 2);
            if (!any_flush) flags |= F_ACC_INIT;
            any_flush = true;
            oldest = k + 2;
        }
        if (last) flags |= F_REDUCE;
        tp.flags = flags;
        tp.reverse = 0;
        ops.push_back(op);
        double2 *oX = X, *oY = Y;
        Y = F1; X = F2; F1 = oX; F2 = oY;
    }
}

// The matrix side of a term launch: everything of TermParams that comes from the handle.
TermParams matrix_params(const tbpm_ham *H, double *partial)
{
    TermParams mp{};
    mp.orp = H->orp; mp.ocol = H->ocol; mp.oidx = H->oidx; mp.vtab = H->vtab; mp.diag = H->diag;
    mp.rowptr = H->rowptr; mp.col = H->col; mp.val = H->val;
    mp.n_orb = H->n_orb;
    mp.partial = partial;
    mp.n_table = H->n_table;
    mp.packed = H->packed;
    mp.single_real = H->single_real;
    mp.device = H->device;
    mp.walk_stride = 0; mp.walk_run = 1;
    mp.n_lat_off = H->n_lat_off;
    for (int j = 0; j < H->n_lat_off; ++j) { mp.lat_off[j] = H->lat_off[j]; mp.lat_delta[j] = H->lat_delta[j]; }
    mp.lat_flags = H->lat_flags;
    mp.n_regular = H->n_regular;
    mp.lat_periodic3 = H->lat_periodic3;
    mp.sq8_line = H->sq8_line; mp.dline = H->dline; mp.sq8_real_x = H->sq8_real_x;
    mp.d16 = H->near16_w > 0 ? H->d16 : nullptr; mp.n16_w = H->near16_w;
    mp.uniform = H->n_orb > 0 && H->min_row_nnz == H->max_row_nnz;
    mp.max_row_off = std::max(0, H->max_row_nnz - (H->has_onsite ? 1 : 0));
    // L2 prefetch of the vector rows a few tiles ahead (term_ph.cuh, producer warp).  The leading edge of the gather
    // window is the farthest neighbour: the largest lattice stride on uniform lattices, else the widest |col - row|.
    mp.pf_dist = knob("pf", 0);
    mp.pf_mask = knob("pf_mask", 3);
    mp.pf_lead = H->n_lat_off > 0 ? H->lat_off[H->n_lat_off - 1] : H->halo_rows;
    if (knob("pf_lead", -1) >= 0) mp.pf_lead = knob("pf_lead", -1);
    return mp;
}

// Two extra vectors of a full tile behind the plan (shared by the tiles, which run one after the other) when the two-terms-per-sweep
// kernel applies to this Hamiltonian; run() falls back to one term per sweep when the caller's workspace lacks them.
size_t pair_extra_bytes(const tbpm_ham *H, const Plan &P)
{
    if (P.tile != 8 || H->n_table <= 0) return 0;
    const TermParams mp = matrix_params(H, nullptr);
    return pair_sq_supported(8, mp) ? 2 * P.full_vec : 0;
}

// Shared body of tbpm_propagate (psi0 != NULL) and tbpm_ldos (sites != NULL).
struct QeSpec { const double *energies; int n_energy; double *out; };   // NEXT-3: energies on the host, out on the device

int run(tbpm_ham *H, const double *psi0, const int64_t *sites, int n_state, int n_step, double dt, double rescale, double *corr,
        double *norm2, void *workspace, size_t workspace_bytes, void *stream, const QeSpec *qe = nullptr)
{
    if (!H || n_state < 0 || n_step < 0 || !(rescale > 0.0) || !(dt >= 0.0) || !std::isfinite(dt) || !std::isfinite(rescale))
        return TBPM_EINVAL;
    const long long launches0 = total_launches();
    H->last_launches = 0;
    if (n_state == 0 || n_step == 0) return TBPM_OK;
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || !corr || (!psi0 && !sites)) return TBPM_EINVAL;
    if (psi0 && (reinterpret_cast<uintptr_t>(psi0) & 15u)) return TBPM_EINVAL;
    if (sites)
        for (int b = 0; b < n_state; ++b)
            if (sites[b] < 0 || sites[b] >= H->n_orb) return TBPM_EINDEX;
    const Plan P = make_plan(H->n_orb, n_state, H->opt_tile);
    const size_t qe_bytes = qe ? (size_t)qe->n_energy * P.full_vec : 0;
    if (workspace_bytes < P.total + qe_bytes) return TBPM_ENOMEM;
    cudaStream_t st = static_cast<cudaStream_t>(stream);

    // a1: coefficients (host, once per call)
    std::vector<double> cf(2 * 8192);
    int K = 0;
    int rc = tbpm_cheb_coeff(rescale * dt, 1e-15, 8192, &K, cf.data());
    if (rc) return rc;

    char *W = static_cast<char *>(workspace);
    double *partial = reinterpret_cast<double *>(W + P.partial_off);
    int64_t *d_sites = reinterpret_cast<int64_t *>(W + P.sites_off);
    if (sites) TBPM_CUDA_TRY(cudaMemcpyAsync(d_sites, sites, sizeof(int64_t) * (size_t)n_state, cudaMemcpyHostToDevice, st));

    // psi sits in slot p_n at the start of step n and moves p -> (p + 2) % 3 every step; start so that it ends in slot 0
    const int start_slot = n_step % 3;

    const bool table = H->n_table > 0;
    TermParams tp = matrix_params(H, partial);
    const bool reverse_odd = knob("rev", 1) != 0;         // odd terms sweep backwards (term_ph.cuh)
    const int kernel_opt = H->opt_kernel;

    std::vector<TermParams> term;
    for (int t = 0; t < P.n_tile; ++t) {
        const int state0 = t * P.tile;
        const int n_valid = std::min(P.tile, n_state - state0);
        const int bt = (t == P.n_tile - 1) ? P.last_bt : P.tile;
        const size_t vec = align_up((size_t)H->n_orb * bt * sizeof(double2));
        char *base = W + P.vec0_off + (size_t)t * 4 * P.full_vec;
        double2 *buf[3] = {reinterpret_cast<double2 *>(base), reinterpret_cast<double2 *>(base + vec),
                           reinterpret_cast<double2 *>(base + 2 * vec)};
        double2 *bra = reinterpret_cast<double2 *>(base + 3 * vec);
        const int64_t n_el = H->n_orb * bt;
        if (n_el > 0) {
            if (psi0) {
                k_interleave<<<(unsigned)((n_el + kThreads - 1) / kThreads), kThreads, 0, st>>>(
                    reinterpret_cast<const double2 *>(psi0), H->n_orb, state0, n_valid, bt, buf[start_slot], bra);
            } else {
                TBPM_CUDA_TRY(cudaMemsetAsync(buf[start_slot], 0, sizeof(double2) * (size_t)n_el, st));
                TBPM_CUDA_TRY(cudaMemsetAsync(bra, 0, sizeof(double2) * (size_t)n_el, st));
                k_unit_states<<<1, kMaxBT, 0, st>>>(d_sites, state0, n_valid, bt, buf[start_slot], bra);
            }
            count_launches(1);
        }
        tp.psi0 = bra;
        int slot = start_slot;
        double2 *qe_ws = reinterpret_cast<double2 *>(W + P.total);   // [n_energy][row][bt] of this tile (NEXT-3)
        const size_t qe_stride = P.full_vec / sizeof(double2);
        const unsigned qe_grid = (unsigned)std::min<int64_t>((n_el + kThreads - 1) / kThreads, (int64_t)H->num_sms * 8);
        auto qe_add = [&](const double2 *psi, int n) {       // qe[e] += w_n exp(+i E_e n dt) psi(n dt), Hann window w_n
            QeCoef cf{};
            const long double wn = 0.5L * (1.0L + cosl(3.14159265358979323846264338327950288L * (long double)n / (long double)n_step));
            for (int e = 0; e < qe->n_energy; ++e) {
                const long double ph = (long double)qe->energies[e] * (long double)n * (long double)dt;
                cf.c[e] = make_double2((double)(wn * cosl(ph)), (double)(wn * sinl(ph)));
            }
            k_qe_axpy<<<qe_grid, kThreads, 0, st>>>(psi, n_el, qe->n_energy, cf, qe_stride, qe_ws, n == 0);
            count_launches(1);
        };
        if (qe && n_el > 0) qe_add(buf[start_slot], 0);
        // two terms per sweep where term_sq2.cu applies (full tiles of 8 states, default kernel choice, room for the two extra vectors)
        const bool pairs = !qe && table && H->opt_kernel == 0 && K >= 3 && bt == 8 && n_el > 0 && pair_sq_supported(bt, tp) &&
                           workspace_bytes >= P.total + 2 * P.full_vec;
        std::vector<StepOp> ops;
        auto one_step = [&](int n, cudaStream_t s2) -> int {
            double2 *psi = buf[slot], *t1 = buf[(slot + 1) % 3], *acc = buf[(slot + 2) % 3];
            int grid = 1;
            if (K == 1) {                                 // tau = 0: psi' = c_0 psi, no H application
                TermParams t0 = tp;
                t0.x = psi; t0.y = t1; t0.acc = acc; t0.a = 0.0;
                t0.ca = make_double2(cf[0], cf[1]); t0.n_acc = 1; t0.flags = F_SKIP_H | F_ACC_INIT | F_REDUCE;
                if ((rc = launch_term(bt, table, 1, t0, H->num_sms, s2, &grid))) return rc;
            }
            if (pairs) {
                step_pairs(tp, K, cf, rescale, psi, t1, acc, reinterpret_cast<double2 *>(W + P.total),
                           reinterpret_cast<double2 *>(W + P.total + P.full_vec), ops);
                for (const StepOp &op : ops)
                    if ((rc = op.pair ? launch_pair_sq(op.tp, H->num_sms, s2, &grid) : launch_term(bt, table, 0, op.tp, H->num_sms, s2, &grid)))
                        return rc;
            } else {
                step_terms(tp, K, cf, rescale, reverse_odd, psi, t1, acc, term);
                for (int k = 1; k < K; ++k)
                    if ((rc = launch_term(bt, table, kernel_opt, term[k], H->num_sms, s2, &grid))) return rc;
            }
            k_reduce_final<<<bt, 96, 0, s2>>>(partial, grid, bt, n_valid, state0, n_step, n, corr, norm2);
            count_launches(1);
            return TBPM_OK;
        };
        // small models: all time steps of the tile in one cluster launch (k_small_steps)
        const bool small = !qe && table && K >= 2 && K <= kSmallMaxK && bt <= 8 && tp.max_row_off <= kSmallCH && n_el > 0 &&
                           n_el <= (int64_t)kSmallRPT * kSmallCluster * kSmallThreads && H->opt_kernel == 0 && knob("small", 1);
        if (small) {
            std::vector<TermLite> all((size_t)3 * K);
            auto which = [&](const double2 *q) { return q == buf[0] ? 0 : (q == buf[1] ? 1 : 2); };
            for (int sl = 0; sl < 3; ++sl) {
                step_terms(tp, K, cf, rescale, false, buf[sl], buf[(sl + 1) % 3], buf[(sl + 2) % 3], term);
                for (int k = 1; k < K; ++k) {
                    const TermParams &q = term[k];
                    all[(size_t)sl * K + k] = TermLite{which(q.x), which(q.y), which(q.acc), q.n_acc, q.flags, q.a, q.ca, q.cb, q.cc};
                }
            }
            TermLite *d_terms = reinterpret_cast<TermLite *>(W + P.aux_off);
            // pageable source: the call returns once the data is staged, so `all` may go out of scope
            TBPM_CUDA_TRY(cudaMemcpyAsync(d_terms, all.data(), all.size() * sizeof(TermLite), cudaMemcpyHostToDevice, st));
            constexpr int kSmallSmem = 4 * kSmallRPT * kSmallThreads * (int)sizeof(double2);   // 128 KB: the most a block can be asked for
            static int cluster_size[kMaxDevices][4] = {};   // per device and tile width: 16 blocks (opt-in cluster size) if they fit, else 8
            const int bi = bt == 1 ? 0 : (bt == 2 ? 1 : (bt == 4 ? 2 : 3));
            if (H->device < 0 || H->device >= kMaxDevices) return TBPM_EINVAL;
            const void *kern = bt == 1 ? (const void *)k_small_steps<1> : bt == 2 ? (const void *)k_small_steps<2> :
                               bt == 4 ? (const void *)k_small_steps<4> : (const void *)k_small_steps<8>;
            cudaLaunchConfig_t cfg{};
            cudaLaunchAttribute attr[1];
            attr[0].id = cudaLaunchAttributeClusterDimension;
            attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
            cfg.blockDim = dim3(kSmallThreads); cfg.stream = st; cfg.attrs = attr; cfg.numAttrs = 1;
            if (cluster_size[H->device][bi] == 0) {
                TBPM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmallSmem));
                int cs = kSmallCluster, n_cl = 0;
                if (cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess) {
                    cfg.gridDim = dim3(kSmallClusterMax); cfg.dynamicSmemBytes = kSmallSmem / 2;
                    attr[0].val.clusterDim.x = kSmallClusterMax;
                    if (cudaOccupancyMaxActiveClusters(&n_cl, kern, &cfg) == cudaSuccess && n_cl >= 1) cs = kSmallClusterMax;
                }
                (void)cudaGetLastError();
                cluster_size[H->device][bi] = cs;
            }
            const int cs = cluster_size[H->device][bi];
            const int E = (int)(((n_el + cs - 1) / cs + bt - 1) / bt * bt);
            SmallParams sp{d_terms, tp.orp, tp.ocol, tp.oidx, tp.vtab, tp.diag, {buf[0], buf[1], buf[2]}, bra, H->n_orb, E, K, n_step,
                           start_slot, n_valid, state0, tp.packed, tp.uniform, tp.max_row_off, corr, norm2, partial};
            cfg.gridDim = dim3(cs); cfg.dynamicSmemBytes = (size_t)4 * E * sizeof(double2);
            attr[0].val.clusterDim.x = cs;
            void *kargs[] = {&sp};
            cudaError_t le = cudaLaunchKernelExC(&cfg, kern, kargs);
            TBPM_CUDA_TRY(le);
            count_launches(1);
            slot = (start_slot + 2 * n_step) % 3;
        }
        for (int n = 0; n < n_step && !small; ++n) {
            if ((rc = one_step(n, st))) return rc;
            slot = (slot + 2) % 3;                        // psi' (acc) is the next step's psi
            if (qe && n_el > 0) qe_add(buf[slot], n + 1);
        }
        if (qe && n_el > 0) {
            k_qe_export<<<qe_grid, kThreads, 0, st>>>(qe_ws, qe_stride, H->n_orb, bt, n_valid, state0, qe->n_energy,
                                                      reinterpret_cast<double2 *>(qe->out));
            count_launches(1);
        }
    }
    TBPM_CUDA_TRY(cudaGetLastError());
    {
        std::lock_guard<std::mutex> lock(H->mu);
        RunRecord rec{workspace, n_state, P.tile, P.last_bt, P.vec0_off, P.full_vec};
        bool found = false;
        for (RunRecord &r : H->runs)
            if (r.workspace == workspace) { r = rec; found = true; }
        if (!found) H->runs.push_back(rec);
    }
    H->last_launches = total_launches() - launches0;
    return TBPM_OK;
}

}  // namespace

extern "C" int tbpm_propagate_bytes(const tbpm_ham *H, int n_state, size_t *workspace_bytes)
{
    if (!H || n_state < 0 || !workspace_bytes) return TBPM_EINVAL;
    const Plan P = make_plan(H->n_orb, n_state, H->opt_tile);
    *workspace_bytes = P.total + pair_extra_bytes(H, P);
    return TBPM_OK;
}

extern "C" int tbpm_propagate(tbpm_ham *H, const double *psi0, int n_state, int n_step, double dt, double rescale, double *corr,
                              double *norm2, void *workspace, size_t workspace_bytes, void *stream)
{
    if (n_state > 0 && n_step > 0 && !psi0) return TBPM_EINVAL;
    return run(H, psi0, nullptr, n_state, n_step, dt, rescale, corr, norm2, workspace, workspace_bytes, stream);
}

extern "C" int tbpm_ldos(tbpm_ham *H, const int64_t *sites, int n_site, int n_step, double dt, double rescale, double *corr,
                         double *norm2, void *workspace, size_t workspace_bytes, void *stream)
{
    if (n_site > 0 && n_step > 0 && !sites) return TBPM_EINVAL;
    return run(H, nullptr, sites, n_site, n_step, dt, rescale, corr, norm2, workspace, workspace_bytes, stream);
}


extern "C" int tbpm_propagate_qe_bytes(const tbpm_ham *H, int n_state, int n_energy, size_t *workspace_bytes)
{
    if (!H || n_state < 0 || n_energy < 0 || n_energy > kMaxEnergy || !workspace_bytes) return TBPM_EINVAL;
    const Plan P = make_plan(H->n_orb, n_state, H->opt_tile);
    *workspace_bytes = P.total + (size_t)n_energy * P.full_vec;
    return TBPM_OK;
}

extern "C" int tbpm_propagate_qe(tbpm_ham *H, const double *psi0, int n_state, int n_step, double dt, double rescale,
                                 const double *energies, int n_energy, double *corr, double *norm2, double *qe, void *workspace,
                                 size_t workspace_bytes, void *stream)
{
    if (n_energy < 0 || n_energy > kMaxEnergy || (n_energy > 0 && (!energies || !qe))) return TBPM_EINVAL;
    if (n_state > 0 && n_step > 0 && !psi0) return TBPM_EINVAL;
    for (int e = 0; e < n_energy; ++e)
        if (!std::isfinite(energies[e])) return TBPM_EINVAL;
    QeSpec spec{energies, n_energy, qe};
    return run(H, psi0, nullptr, n_state, n_step, dt, rescale, corr, norm2, workspace, workspace_bytes, stream, n_energy > 0 ? &spec : nullptr);
}

// NEXT-2: Haydock recursion from the given sites.  Workspace = that of tbpm_propagate for n_site states (three rotating vectors
// per tile are enough; the fourth holds nothing here).
extern "C" int tbpm_haydock(tbpm_ham *H, const int64_t *sites, int n_site, int n_iter, double *a_out, double *b_out, void *workspace,
                            size_t workspace_bytes, void *stream)
{
    if (!H || n_site < 0 || n_iter < 0) return TBPM_EINVAL;
    if (n_site == 0 || n_iter == 0) return TBPM_OK;
    if (!sites || !a_out || !b_out || !workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u)) return TBPM_EINVAL;
    for (int b = 0; b < n_site; ++b)
        if (sites[b] < 0 || sites[b] >= H->n_orb) return TBPM_EINDEX;
    const Plan P = make_plan(H->n_orb, n_site, H->opt_tile);
    if (workspace_bytes < P.total) return TBPM_ENOMEM;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    char *W = static_cast<char *>(workspace);
    double *partial = reinterpret_cast<double *>(W + P.partial_off);
    double *sc = reinterpret_cast<double *>(W + P.aux_off);   // [bt][4] scalars, then [nn_grid][bt] norm partials
    double *nn_partial = sc + 4 * kMaxBT;
    int64_t *d_sites = reinterpret_cast<int64_t *>(W + P.sites_off);
    TBPM_CUDA_TRY(cudaMemcpyAsync(d_sites, sites, sizeof(int64_t) * (size_t)n_site, cudaMemcpyHostToDevice, st));
    const bool table = H->n_table > 0;
    TermParams tp = matrix_params(H, partial);
    // t = H u_n and <u_n|t> in one sweep: the last-term shape of the fused kernel with psi' := 1 * T_k, first flush, bra = u_n
    tp.a = 1.0; tp.ca = make_double2(1.0, 0.0); tp.n_acc = 1; tp.flags = F_ACC_INIT | F_REDUCE;
    const int nn_grid = std::max(1, std::min(H->num_sms * 8, (int)((kAuxBytes / sizeof(double) - 4 * kMaxBT) / kMaxBT)));   // norm partials: [nn_grid][bt] doubles in the aux area
    int rc = TBPM_OK;
    for (int t = 0; t < P.n_tile; ++t) {
        const int state0 = t * P.tile;
        const int n_valid = std::min(P.tile, n_site - state0);
        const int bt = (t == P.n_tile - 1) ? P.last_bt : P.tile;
        const size_t vec = align_up((size_t)H->n_orb * bt * sizeof(double2));
        char *base = W + P.vec0_off + (size_t)t * 4 * P.full_vec;
        double2 *u = reinterpret_cast<double2 *>(base), *u_prev = reinterpret_cast<double2 *>(base + vec),
                *tv = reinterpret_cast<double2 *>(base + 2 * vec);
        const int64_t n_el = H->n_orb * bt;
        TBPM_CUDA_TRY(cudaMemsetAsync(u, 0, sizeof(double2) * (size_t)n_el, st));
        TBPM_CUDA_TRY(cudaMemsetAsync(u_prev, 0, sizeof(double2) * (size_t)n_el, st));
        k_unit_states<<<1, kMaxBT, 0, st>>>(d_sites, state0, n_valid, bt, u, u);
        k_haydock_init<<<1, kMaxBT, 0, st>>>(sc, bt, n_valid);
        count_launches(2);
        for (int it = 0; it < n_iter; ++it) {
            int grid = 1;
            tp.x = u; tp.psi0 = u; tp.acc = tv; tp.y = u_prev;    // y is neither read nor written by this shape
            if ((rc = launch_term(bt, table, H->opt_kernel, tp, H->num_sms, st, &grid))) return rc;
            k_haydock_scalars<<<bt, 32, 0, st>>>(partial, grid, bt, sc, 0, nn_partial, nn_grid, n_valid, state0, n_iter, it, a_out, b_out);
            k_haydock_update<<<nn_grid, 256, 0, st>>>(tv, u, u_prev, H->n_orb, bt, sc, nn_partial);
            k_haydock_scalars<<<bt, 32, 0, st>>>(partial, grid, bt, sc, 1, nn_partial, nn_grid, n_valid, state0, n_iter, it, a_out, b_out);
            count_launches(3);
            std::swap(u, u_prev);                             // u_{n+1} was written over u_{n-1}
        }
    }
    TBPM_CUDA_TRY(cudaGetLastError());
    return TBPM_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// NEXT-4: AC-conductivity correlation  corr[b][n] = < psi2(n dt) | J_a | psi1(n dt) >,  psi1(0) = [1 - f(H)] J_b psi0,
// psi2(0) = f(H) psi0  (reading #30).  Everything runs on the fused term kernels: a Chebyshev series (Fermi operator or
// time step) is K - 1 term launches with the series' coefficients, J x is the first-term shape with J's matrix, and
// <psi2|J_a psi1> is the last-term shape (first flush of 1 * T, bra = psi2) with J_a's matrix.  One tile of states at a time:
// two sets of three rotating vectors.
// ---------------------------------------------------------------------------------------------------------------------
extern "C" int tbpm_corr_ac_bytes(const tbpm_ham *H, int n_state, size_t *workspace_bytes)
{
    if (!H || n_state < 0 || !workspace_bytes) return TBPM_EINVAL;
    const Plan P = make_plan(H->n_orb, n_state, H->opt_tile);
    *workspace_bytes = P.vec0_off + 6 * P.full_vec + pair_extra_bytes(H, P);   // + two vectors where two terms per sweep apply
    return TBPM_OK;
}

namespace {
// The two operators are either matrices (Ja, Jb: current operators) or diagonals (da, db: density operators, device [n_orb][2]).
int corr_pair(tbpm_ham *H, tbpm_ham *Ja, tbpm_ham *Jb, const double2 *da, const double2 *db, const double *psi0, int n_state, int n_step,
              double dt, double rescale, double beta, double mu, double *corr, void *workspace, size_t workspace_bytes, void *stream)
{
    const bool diag_op = da != nullptr;
    if (diag_op) { Ja = H; Jb = H; }                     // placeholders: the matrix launches below are not used
    if (!H || !Ja || !Jb || n_state < 0 || n_step < 0 || !(rescale > 0.0) || !(dt >= 0.0) || !std::isfinite(dt) || !std::isfinite(rescale))
        return TBPM_EINVAL;
    if (Ja->n_orb != H->n_orb || Jb->n_orb != H->n_orb || Ja->device != H->device || Jb->device != H->device) return TBPM_EINVAL;
    if (n_state == 0) return TBPM_OK;
    if (!psi0 || !corr || !workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || (reinterpret_cast<uintptr_t>(psi0) & 15u)) return TBPM_EINVAL;
    const Plan P = make_plan(H->n_orb, n_state, H->opt_tile);
    if (workspace_bytes < P.vec0_off + 6 * P.full_vec) return TBPM_ENOMEM;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const long long launches0 = total_launches();

    std::vector<double> ct(2 * 8192), cf(2 * 8192), cg(2 * 8192);   // time step, f, 1 - f
    int Kt = 0, Kf = 0, Kg = 0, rc;
    if ((rc = tbpm_cheb_coeff(rescale * dt, 1e-15, 8192, &Kt, ct.data()))) return rc;
    if ((rc = tbpm_fermi_coeff(beta, mu, rescale, 0, 1e-13, 8192, &Kf, cf.data()))) return rc;
    if ((rc = tbpm_fermi_coeff(beta, mu, rescale, 1, 1e-13, 8192, &Kg, cg.data()))) return rc;

    char *W = static_cast<char *>(workspace);
    double *partial = reinterpret_cast<double *>(W + P.partial_off);
    const TermParams mh = matrix_params(H, partial), ma = matrix_params(Ja, partial), mb = matrix_params(Jb, partial);
    const bool reverse_odd = knob("rev", 1) != 0;
    std::vector<TermParams> term;
    const int n_out = n_step + 1;

    for (int t = 0; t < P.n_tile; ++t) {
        const int state0 = t * P.tile;
        const int n_valid = std::min(P.tile, n_state - state0);
        const int bt = (t == P.n_tile - 1) ? P.last_bt : P.tile;
        const size_t vec = align_up((size_t)H->n_orb * bt * sizeof(double2));
        char *base = W + P.vec0_off;
        double2 *A[3], *B[3];
        for (int i = 0; i < 3; ++i) { A[i] = reinterpret_cast<double2 *>(base + i * vec); B[i] = reinterpret_cast<double2 *>(base + (3 + i) * vec); }
        const int64_t n_el = H->n_orb * bt;
        if (n_el == 0) continue;
        k_interleave<<<(unsigned)((n_el + kThreads - 1) / kThreads), kThreads, 0, st>>>(reinterpret_cast<const double2 *>(psi0), H->n_orb, state0,
                                                                                       n_valid, bt, A[0], B[0]);
        count_launches(1);
        int grid = 1;
        // two terms per sweep where term_sq2.cu applies and the caller's workspace holds the two extra vectors (behind the six)
        const bool pairs = H->n_table > 0 && H->opt_kernel == 0 && bt == 8 && pair_sq_supported(bt, mh) &&
                           workspace_bytes >= P.vec0_off + 8 * P.full_vec;
        double2 *e1 = reinterpret_cast<double2 *>(base + 6 * P.full_vec), *e2 = reinterpret_cast<double2 *>(base + 7 * P.full_vec);
        std::vector<StepOp> ops;
        // a Chebyshev series sum_k c_k T_k(H / s) applied to buf[slot]; returns the slot that holds the result
        auto series = [&](double2 **buf, int slot, int K, const std::vector<double> &c) -> int {
            double2 *psi = buf[slot], *t1 = buf[(slot + 1) % 3], *acc = buf[(slot + 2) % 3];
            TermParams tp = mh;
            tp.psi0 = psi;                                // the last term's dot products are not used here
            if (pairs && K >= 3) {
                step_pairs(tp, K, c, rescale, psi, t1, acc, e1, e2, ops);
                for (size_t o = 0; o < ops.size() && !rc; ++o)
                    rc = ops[o].pair ? launch_pair_sq(ops[o].tp, H->num_sms, st, &grid) : launch_term(bt, true, 0, ops[o].tp, H->num_sms, st, &grid);
                return (slot + 2) % 3;
            }
            if (K == 1) {
                TermParams t0 = tp;
                t0.x = psi; t0.y = t1; t0.acc = acc; t0.a = 0.0;
                t0.ca = make_double2(c[0], c[1]); t0.n_acc = 1; t0.flags = F_SKIP_H | F_ACC_INIT | F_REDUCE;
                rc = launch_term(bt, H->n_table > 0, 1, t0, H->num_sms, st, &grid);
            } else {
                step_terms(tp, K, c, rescale, reverse_odd, psi, t1, acc, term);
                for (int k = 1; k < K && !rc; ++k) rc = launch_term(bt, H->n_table > 0, H->opt_kernel, term[k], H->num_sms, st, &grid);
            }
            return (slot + 2) % 3;
        };
        // corr[.][n] = <psi2|J_a psi1>: J_a psi1 goes to a free buffer of set A
        const int dgrid = (int)std::min<int64_t>((n_el + 255) / 256, (int64_t)H->num_sms * 8);
        auto cross = [&](int sa, int sb, int n) {
            if (diag_op) {
                switch (bt) {
                case 1: k_diag_dot<1><<<dgrid, 256, 0, st>>>(da, A[sa], B[sb], H->n_orb, partial); break;
                case 2: k_diag_dot<2><<<dgrid, 256, 0, st>>>(da, A[sa], B[sb], H->n_orb, partial); break;
                case 4: k_diag_dot<4><<<dgrid, 256, 0, st>>>(da, A[sa], B[sb], H->n_orb, partial); break;
                case 8: k_diag_dot<8><<<dgrid, 256, 0, st>>>(da, A[sa], B[sb], H->n_orb, partial); break;
                case 16: k_diag_dot<16><<<dgrid, 256, 0, st>>>(da, A[sa], B[sb], H->n_orb, partial); break;
                default: k_diag_dot<32><<<dgrid, 256, 0, st>>>(da, A[sa], B[sb], H->n_orb, partial); break;
                }
                k_reduce_final<<<bt, 96, 0, st>>>(partial, dgrid, bt, n_valid, state0, n_out, n, corr, nullptr);
                count_launches(2);
                return;
            }
            TermParams tp = ma;
            tp.x = A[sa]; tp.psi0 = B[sb]; tp.acc = A[(sa + 1) % 3]; tp.y = A[(sa + 2) % 3];
            tp.a = 1.0; tp.ca = make_double2(1.0, 0.0); tp.n_acc = 1; tp.flags = F_ACC_INIT | F_REDUCE;
            rc = launch_term(bt, Ja->n_table > 0, Ja->opt_kernel, tp, Ja->num_sms, st, &grid);
            k_reduce_final<<<bt, 96, 0, st>>>(partial, grid, bt, n_valid, state0, n_out, n, corr, nullptr);
            count_launches(1);
        };
        rc = TBPM_OK;
        if (diag_op) {                                    // A[1] = d_b psi0
            k_diag_apply<<<dgrid, 256, 0, st>>>(db, A[0], A[1], H->n_orb, bt);
            count_launches(1);
        } else {                                          // A[1] = J_b psi0 (first-term shape: y = a J x)
            TermParams tp = mb;
            tp.x = A[0]; tp.y = A[1]; tp.acc = A[2]; tp.psi0 = A[0];
            tp.a = 1.0; tp.n_acc = 0; tp.flags = F_WRITE_Y;
            rc = launch_term(bt, Jb->n_table > 0, Jb->opt_kernel, tp, Jb->num_sms, st, &grid);
        }
        if (rc) return rc;
        int sa = series(A, 1, Kg, cg);                    // psi1 = [1 - f(H)] J_b psi0
        if (rc) return rc;
        int sb = series(B, 0, Kf, cf);                    // psi2 = f(H) psi0
        if (rc) return rc;
        cross(sa, sb, 0);
        for (int n = 1; n <= n_step && !rc; ++n) {
            sa = series(A, sa, Kt, ct);
            if (!rc) sb = series(B, sb, Kt, ct);
            if (!rc) cross(sa, sb, n);
        }
        if (rc) return rc;
    }
    TBPM_CUDA_TRY(cudaGetLastError());
    H->last_launches = total_launches() - launches0;
    return TBPM_OK;
}
}  // namespace

extern "C" int tbpm_corr_ac(tbpm_ham *H, tbpm_ham *Ja, tbpm_ham *Jb, const double *psi0, int n_state, int n_step, double dt, double rescale,
                            double beta, double mu, double *corr, void *workspace, size_t workspace_bytes, void *stream)
{
    if (!Ja || !Jb) return TBPM_EINVAL;
    return corr_pair(H, Ja, Jb, nullptr, nullptr, psi0, n_state, n_step, dt, rescale, beta, mu, corr, workspace, workspace_bytes, stream);
}

extern "C" int tbpm_corr_dp(tbpm_ham *H, const double *rho_a, const double *rho_b, const double *psi0, int n_state, int n_step, double dt,
                            double rescale, double beta, double mu, double *corr, void *workspace, size_t workspace_bytes, void *stream)
{
    if (!rho_a || !rho_b || (reinterpret_cast<uintptr_t>(rho_a) & 15u) || (reinterpret_cast<uintptr_t>(rho_b) & 15u)) return TBPM_EINVAL;
    return corr_pair(H, nullptr, nullptr, reinterpret_cast<const double2 *>(rho_a), reinterpret_cast<const double2 *>(rho_b), psi0, n_state, n_step,
                     dt, rescale, beta, mu, corr, workspace, workspace_bytes, stream);
}

extern "C" int tbpm_get_state(const tbpm_ham *H, const void *workspace, int state, double *psi_out, void *stream)
{
    if (!H || !workspace || !psi_out || state < 0) return TBPM_EINVAL;
    RunRecord rec{};
    {
        std::lock_guard<std::mutex> lock(H->mu);
        bool found = false;
        for (const RunRecord &r : H->runs)
            if (r.workspace == workspace) { rec = r; found = true; }
        if (!found) return TBPM_EINVAL;                   // no tbpm_propagate / tbpm_ldos call of this handle used that workspace
    }
    if (state >= rec.n_state) return TBPM_EINDEX;
    if (H->n_orb == 0) return TBPM_OK;
    const int tile = state / rec.tile;
    const int n_tile = (rec.n_state + rec.tile - 1) / rec.tile;
    const int bt = (tile == n_tile - 1) ? rec.last_bt : rec.tile;
    // psi ends in slot 0 of its tile's buffers (run() starts it in slot n_step % 3)
    const double2 *psi = reinterpret_cast<const double2 *>(static_cast<const char *>(workspace) + rec.vec0_off + (size_t)tile * 4 * rec.full_vec);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int grid = (int)std::min<int64_t>((H->n_orb + kThreads - 1) / kThreads, 4096);
    k_get_state<<<grid, kThreads, 0, st>>>(psi, H->n_orb, bt, state - tile * rec.tile, reinterpret_cast<double2 *>(psi_out));
    count_launches(1);
    TBPM_CUDA_TRY(cudaGetLastError());
    return TBPM_OK;
}

extern "C" int64_t tbpm_last_launch_count(const tbpm_ham *H) { return H ? (int64_t)H->last_launches : 0; }

extern "C" int tbpm_set_option(tbpm_ham *H, int option, int64_t value)
{
    if (!H) return TBPM_EINVAL;
    switch (option) {
    case TBPM_OPT_TILE:
        if (value != 1 && value != 2 && value != 4 && value != 8 && value != 16 && value != 32) return TBPM_EINVAL;
        H->opt_tile = (int)value;
        return TBPM_OK;
    case TBPM_OPT_KERNEL:
        if (value < 0 || value > 4) return TBPM_EINVAL;
        H->opt_kernel = (int)value;
        return TBPM_OK;
    }
    return TBPM_EINVAL;
}

// ---------------------------------------------------------------------------------------------------------------------
// tbpm_propagate_static: the same propagation with NO caller workspace and NO allocation of any kind
// ---------------------------------------------------------------------------------------------------------------------
// For callers that cannot allocate device memory (CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): the
// workspace of tbpm_propagate -- block partials of the fused dot products, term descriptors, and the four vectors per state tile --
// lives in ONE file-scope device array of TBPM_STATIC_WORKSPACE_BYTES.  Every GPU that loads the library holds the array until the
// process exits.  All calls on a device share it and it keeps the previous call's contents: run() initialises everything it reads
// (it is written for uninitialised workspaces), but two calls that overlap on the GPU (different streams, or host threads) RACE.
static __device__ __align__(256) unsigned char g_static_workspace[TBPM_STATIC_WORKSPACE_BYTES];

namespace {
std::mutex g_static_mu;
void *g_static_ptr[kMaxDevices] = {nullptr};   // device address of g_static_workspace per device (in host code the symbol is only a stand-in)
}  // namespace

extern "C" int tbpm_propagate_static(tbpm_ham *H, const double *psi0, int n_state, int n_step, double dt, double rescale, double *corr,
                                     double *norm2, void *stream)
{
    if (!H || n_state < 0 || n_step < 0) return TBPM_EINVAL;
    if (n_state == 0 || n_step == 0) return TBPM_OK;        // as in tbpm_propagate: success, outputs untouched
    if (!psi0) return TBPM_EINVAL;
    const size_t need = make_plan(H->n_orb, n_state, H->opt_tile).total;
    if (need > (size_t)TBPM_STATIC_WORKSPACE_BYTES) return TBPM_ETOOBIG;
    int dev = -1;
    TBPM_CUDA_TRY(cudaGetDevice(&dev));
    if (dev != H->device || dev < 0 || dev >= kMaxDevices) return TBPM_EINVAL;   // the array of the CURRENT device is the one addressed
    void *ws = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_static_mu);
        if (!g_static_ptr[dev]) {                           // once per device, with that device current
            void *p = nullptr;
            TBPM_CUDA_TRY(cudaGetSymbolAddress(&p, g_static_workspace));
            g_static_ptr[dev] = p;
        }
        ws = g_static_ptr[dev];
    }
    return run(H, psi0, nullptr, n_state, n_step, dt, rescale, corr, norm2, ws, (size_t)TBPM_STATIC_WORKSPACE_BYTES, stream);
}

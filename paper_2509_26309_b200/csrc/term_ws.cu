// term_ws.cu -- the hot kernel: warp-specialised, bulk-copy (TMA) staged fused Chebyshev term (kernel layout only).
//
//   T_k = a*H*T_{k-1} - T_{k-2}  (amxsy)  fused with  psi' += sum c_j T_j  (axpy, up to
//   three terms at once) and, on the last term of a time step, <psi0|psi'> and <psi'|psi'> (calc_corr_dos).
//
//   producer warp (one elected lane): for every tile of R rows, kept n_stage tiles ahead of the compute, issues 1-D bulk
//       copies (cp.async.bulk + mbarrier complete_tx; SASS UBLKCP) of the tile's row offsets, column indices, value
//       indices, diagonal slice and y / psi' / psi0 slices into a shared-memory stage;
//   8 consumer warps: wait on the stage's "full" mbarrier; per non-zero the dependent chain is ONE deep (index from
//       shared memory -> gather x[col] with a 128/256-bit LDG through L1/L2 -> complex FMA); results go straight to
//       global memory; each warp then arrives on the stage's "empty" mbarrier.  No block-wide barrier in the main loop.
//
// Thread -> (row, SPT consecutive states); SPT = 2 (one LDG.E.256 per gather) when the tile has >= 2 states.
// What varies per term (accumulate 0..3 terms, reduce or not) is a template parameter so that the inner loop carries no
// flag tests; what varies rarely (first term, first flush, diagonal present) is a warp-uniform runtime predicate.
#include <algorithm>

#include "term.h"

namespace tbpm_detail {
namespace {

constexpr int kTabSmem = 256;            // hopping-value tables up to this size are copied into shared memory
constexpr int kConsumers = 256;          // 8 consumer warps
constexpr int kWsThreads = kConsumers + 32;
constexpr int kMaxStages = 8;

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cta.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src), "r"(bytes),
                 "r"(bar)
                 : "memory");
}

// SPT consecutive complex128 values of one row
template <int SPT> struct CVec;
template <> struct CVec<1> {
    double2 v[1];
    __device__ __forceinline__ void ldg(const double2 *p) { v[0] = __ldg(p); }
    __device__ __forceinline__ void lds(const double2 *p) { v[0] = *p; }
    __device__ __forceinline__ void st(double2 *p) const { *p = v[0]; }
    __device__ __forceinline__ void st_cs(double2 *p) const { __stcs(p, v[0]); }
};
template <> struct CVec<2> {
    double2 v[2];
    __device__ __forceinline__ void ldg(const double2 *p)     // one 256-bit load (LDG.E.256)
    {
        asm("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(v[0].x), "=d"(v[0].y), "=d"(v[1].x), "=d"(v[1].y) : "l"(p));
    }
    __device__ __forceinline__ void lds(const double2 *p) { v[0] = p[0]; v[1] = p[1]; }
    __device__ __forceinline__ void st(double2 *p) const
    {
        asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(v[0].x), "d"(v[0].y), "d"(v[1].x), "d"(v[1].y) : "memory");
    }
    __device__ __forceinline__ void st_cs(double2 *p) const
    {
        asm volatile("st.global.cs.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(v[0].x), "d"(v[0].y), "d"(v[1].x), "d"(v[1].y) : "memory");
    }
};

// NACC: terms added to psi' by this launch (0..3); REDUCE: last term of the time step (dot products, T_k not stored);
// T2: the hopping-value table has <= 2 entries and lives in registers.
template <int BT, int NACC, bool REDUCE, bool T2>
__global__ void __launch_bounds__(kWsThreads, 3) k_term_ws(const TermParams p)
{
    constexpr int SPT = BT >= 2 ? 2 : 1;
    constexpr int LPR = BT / SPT;                           // lanes per row
    constexpr int R = kConsumers / LPR;                     // rows per tile
    constexpr uint32_t kVecBytes = R * BT * sizeof(double2);
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t bars[2 * kMaxStages];  // [0, S): full, [kMaxStages, kMaxStages + S): empty
    __shared__ uint32_t lo_s[kMaxStages][2];                // first column / value-index element held by each stage
    __shared__ double2 tab_s[T2 ? 1 : kTabSmem];
    __shared__ double red_s[REDUCE ? kConsumers / 32 : 1][kMaxBT][3];

    const int tid = threadIdx.x;
    const bool sub_y = p.flags & F_SUB_Y;
    const bool need_y = sub_y || NACC == 3;
    const bool need_acc = NACC > 0 && !(p.flags & F_ACC_INIT);
    const bool has_diag = p.diag != nullptr;
    const bool tab_in_smem = !T2 && p.n_table <= kTabSmem;
    const int S = p.n_stage;
    const int64_t n_tiles = (p.n_orb + R - 1) / R;
    const int slot_acc = need_y ? 1 : 0, slot_z = slot_acc + (need_acc ? 1 : 0);   // y is slot 0
    const uint32_t bar0 = smem_u32(bars), smem0 = smem_u32(smem);

    if (tid == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(bar0 + 8 * s, 1); mbar_init(bar0 + 8 * (kMaxStages + s), kConsumers / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (tab_in_smem)
        for (int i = tid; i < p.n_table; i += kWsThreads) tab_s[i] = __ldg(p.vtab + i);
    __syncthreads();

    if (tid >= kConsumers) {
        // ------------------------------------------------ producer warp ------------------------------------------------
        if (tid != kConsumers) return;
        uint32_t q_lo = 0, q_hi = 0;                        // offsets bounding the next tile to issue (prefetched)
        int64_t tile = blockIdx.x;
        if (tile < n_tiles) {
            const int64_t r0 = tile * R;
            q_lo = __ldg(p.orp + r0);
            q_hi = __ldg(p.orp + min(r0 + R, p.n_orb));
        }
        int s = 0;
        uint32_t ph = 1;                                    // parity of the "empty" phase to wait for; first pass: free
        for (; tile < n_tiles; tile += gridDim.x) {
            const uint32_t c_lo = q_lo, c_hi = q_hi;
            const int64_t nt = tile + gridDim.x;
            if (nt < n_tiles) {                             // bounds of the following tile: latency hidden behind this issue
                const int64_t nr0 = nt * R;
                q_lo = __ldg(p.orp + nr0);
                q_hi = __ldg(p.orp + min(nr0 + R, p.n_orb));
            }
            const uint32_t full = bar0 + 8 * s;
            mbar_wait(bar0 + 8 * (kMaxStages + s), ph);     // a fresh barrier reports the "previous" phase complete
            const uint32_t st = smem0 + (uint32_t)s * (uint32_t)p.stage_bytes;
            const int64_t r0 = tile * R;
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
                bulk_g2s(st + p.off_idx, p.oidx + idx_lo, ni * 2, full);
                tx += nc * 4 + ni * 2;
            }
            if (has_diag) {
                const uint32_t db = (uint32_t)((rows * 8 + 15) & ~15);
                bulk_g2s(st + p.off_diag, p.diag + r0, db, full);
                tx += db;
            }
            const uint32_t vb = (uint32_t)rows * BT * sizeof(double2);
            const uint32_t vec = st + p.off_vec;
            const int64_t e0 = r0 * BT;
            if (need_y) { bulk_g2s(vec, p.y + e0, vb, full); tx += vb; }
            if (need_acc) { bulk_g2s(vec + slot_acc * kVecBytes, p.acc + e0, vb, full); tx += vb; }
            if (REDUCE) { bulk_g2s(vec + slot_z * kVecBytes, p.psi0 + e0, vb, full); tx += vb; }
            mbar_expect_tx(full, tx);                       // release: also publishes lo_s[s]
            if (++s == S) { s = 0; ph ^= 1u; }
        }
        return;
    }

    // ---------------------------------------------------- consumer warps ----------------------------------------------------
    const int rl = tid / LPR;                               // row within the tile
    const int b0 = (tid % LPR) * SPT;                       // first state of this thread
    const double2 *xb = p.x + b0;
    const int le = rl * BT + b0;                            // element within a vector slice of the stage
    double2 t0 = make_double2(0.0, 0.0), t1 = t0;           // T2: the one hopping value and its conjugate, in registers
    if (T2) {
        t0 = __ldg(p.vtab);
        t1 = make_double2(t0.x, -t0.y);                     // the one table value and its conjugate
    }
    double s_re[SPT], s_im[SPT], s_nn[SPT];
#pragma unroll
    for (int k = 0; k < SPT; ++k) s_re[k] = s_im[k] = s_nn[k] = 0.0;

    int s = 0;
    uint32_t ph = 0;
    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        mbar_wait(bar0 + 8 * s, ph);
        const unsigned char *st = smem + (size_t)s * p.stage_bytes;
        const int64_t row = tile * R + rl;
        if (row < p.n_orb) {
            const int64_t e = row * BT + b0;
            const double2 *vec = reinterpret_cast<const double2 *>(st + p.off_vec);
            CVec<SPT> xrow, h;
#pragma unroll
            for (int k = 0; k < SPT; ++k) h.v[k] = xrow.v[k] = make_double2(0.0, 0.0);
            if (NACC >= 2 || has_diag) xrow.ldg(p.x + e);   // the tile's own x rows are gathered by its neighbours: L1 hit
            const uint32_t *orp_s = reinterpret_cast<const uint32_t *>(st);
            const uint32_t q0 = orp_s[rl], n = orp_s[rl + 1] - q0;
            const int32_t *cs = reinterpret_cast<const int32_t *>(st + p.off_col) + (q0 - lo_s[s][0]);
            const uint16_t *is = reinterpret_cast<const uint16_t *>(st + p.off_idx) + (q0 - lo_s[s][1]);
            auto value = [&](uint32_t i) -> double2 {
                if (T2) return i ? t1 : t0;
                return table_value(tab_in_smem ? tab_s[i & 0x7fffu] : __ldg(p.vtab + (i & 0x7fffu)), i);
            };
            for (uint32_t j = 0; j < n; j += 4) {           // up to 4 independent gathers in flight, predicated tail
                const bool p1 = j + 1 < n, p2 = j + 2 < n, p3 = j + 3 < n;
                CVec<SPT> x0, x1, x2, x3;
#pragma unroll
                for (int k = 0; k < SPT; ++k) x1.v[k] = x2.v[k] = x3.v[k] = make_double2(0.0, 0.0);
                x0.ldg(xb + (int64_t)(cs[j] & 0x7fffffff) * BT);
                if (p1) x1.ldg(xb + (int64_t)(cs[j + 1] & 0x7fffffff) * BT);
                if (p2) x2.ldg(xb + (int64_t)(cs[j + 2] & 0x7fffffff) * BT);
                if (p3) x3.ldg(xb + (int64_t)(cs[j + 3] & 0x7fffffff) * BT);
                const double2 v0 = value(is[j]);
                const double2 v1 = value(p1 ? is[j + 1] : 0), v2 = value(p2 ? is[j + 2] : 0), v3 = value(p3 ? is[j + 3] : 0);
#pragma unroll
                for (int k = 0; k < SPT; ++k) {             // x1..x3 are zero where the slot is past the row end
                    cfma(h.v[k], v0, x0.v[k]);
                    cfma(h.v[k], v1, x1.v[k]);
                    cfma(h.v[k], v2, x2.v[k]);
                    cfma(h.v[k], v3, x3.v[k]);
                }
            }
            if (has_diag) {
                const double d = reinterpret_cast<const double *>(st + p.off_diag)[rl];
#pragma unroll
                for (int k = 0; k < SPT; ++k) { h.v[k].x = fma(d, xrow.v[k].x, h.v[k].x); h.v[k].y = fma(d, xrow.v[k].y, h.v[k].y); }
            }
#pragma unroll
            for (int k = 0; k < SPT; ++k) { h.v[k].x *= p.a; h.v[k].y *= p.a; }
            CVec<SPT> yold;
#pragma unroll
            for (int k = 0; k < SPT; ++k) yold.v[k] = make_double2(0.0, 0.0);
            if (need_y) yold.lds(vec + le);
            if (sub_y) {
#pragma unroll
                for (int k = 0; k < SPT; ++k) { h.v[k].x -= yold.v[k].x; h.v[k].y -= yold.v[k].y; }
            }
            if (!REDUCE) h.st(p.y + e);                     // T_k: gathered by the next term, keep it cacheable
            if (NACC > 0) {
                CVec<SPT> sacc;
#pragma unroll
                for (int k = 0; k < SPT; ++k) sacc.v[k] = make_double2(0.0, 0.0);
                if (need_acc) sacc.lds(vec + slot_acc * (R * BT) + le);
#pragma unroll
                for (int k = 0; k < SPT; ++k) {
                    cfma(sacc.v[k], p.ca, h.v[k]);
                    if (NACC >= 2) cfma(sacc.v[k], p.cb, xrow.v[k]);
                    if (NACC == 3) cfma(sacc.v[k], p.cc, yold.v[k]);
                }
                if (REDUCE) {
                    CVec<SPT> z;
                    z.lds(vec + slot_z * (R * BT) + le);
#pragma unroll
                    for (int k = 0; k < SPT; ++k) {
                        s_re[k] = fma(z.v[k].x, sacc.v[k].x, s_re[k]);      // conj(z) * psi'
                        s_re[k] = fma(z.v[k].y, sacc.v[k].y, s_re[k]);
                        s_im[k] = fma(z.v[k].x, sacc.v[k].y, s_im[k]);
                        s_im[k] = fma(-z.v[k].y, sacc.v[k].x, s_im[k]);
                        s_nn[k] = fma(sacc.v[k].x, sacc.v[k].x, s_nn[k]);
                        s_nn[k] = fma(sacc.v[k].y, sacc.v[k].y, s_nn[k]);
                    }
                    sacc.st(p.acc + e);                     // psi': T_0 of the next step, gathered right away
                } else {
                    sacc.st_cs(p.acc + e);
                }
            }
        }
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(bar0 + 8 * (kMaxStages + s));   // this warp is done with stage s
        if (++s == S) { s = 0; ph ^= 1u; }
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

template <int BT, int NACC, bool REDUCE, bool T2>
int launch_one(TermParams p, int num_sms, cudaStream_t st, int *grid_out)
{
    constexpr int SPT = BT >= 2 ? 2 : 1;
    constexpr int R = kConsumers / (BT / SPT);
    const bool need_y = (p.flags & F_SUB_Y) || NACC == 3;
    const bool need_acc = NACC > 0 && !(p.flags & F_ACC_INIT);
    const int nvec = (need_y ? 1 : 0) + (need_acc ? 1 : 0) + (REDUCE ? 1 : 0);
    p.n_stage = std::min(kMaxStages, std::max(2, env_int("TBPM_STAGES", 3)));
    p.cap_entries = ((R * std::max(p.max_row_off, 1) + 8 + 7) / 8) * 8;          // + alignment slack of the slice start
    size_t o = (size_t)(((R + 1) * 4 + 15) & ~15);
    p.off_col = (int)o;  o += (size_t)p.cap_entries * 4;
    p.off_idx = (int)o;  o += (size_t)p.cap_entries * 2;
    o = (o + 15) & ~size_t(15);
    p.off_diag = (int)o; o += (size_t)((R * 8 + 15) & ~15);
    o = (o + 127) & ~size_t(127);
    p.off_vec = (int)o;  o += (size_t)nvec * R * BT * sizeof(double2);
    p.stage_bytes = (int)((o + 127) & ~size_t(127));
    const size_t dyn = (size_t)p.stage_bytes * p.n_stage;
    auto kern = k_term_ws<BT, NACC, REDUCE, T2>;
    static size_t configured = 0;
    static int cached_nb = 0;
    static size_t cached_dyn = 0;
    if (dyn > configured) {
        const size_t want = std::max(dyn, (size_t)64 * 1024);
        TBPM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)want));
        configured = want;
    }
    if (cached_dyn != dyn || cached_nb == 0) {
        int nb = 0;
        TBPM_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, kWsThreads, dyn));
        if (nb < 1) return TBPM_ENOMEM;
        cached_nb = nb;
        cached_dyn = dyn;
    }
    const int nb = std::min(cached_nb, std::max(1, env_int("TBPM_MAXB", 8)));
    const int64_t need = (p.n_orb + R - 1) / R;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>({need, (int64_t)num_sms * nb, (int64_t)kMaxGrid}));
    kern<<<grid, kWsThreads, dyn, st>>>(p);
    count_launches(1);
    *grid_out = grid;
    return TBPM_OK;
}

template <int BT, bool T2>
int launch_variant(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    const bool red = p.flags & F_REDUCE;
    if (!red && p.n_acc == 0) return launch_one<BT, 0, false, T2>(p, num_sms, st, grid_out);
    if (!red && p.n_acc == 3) return launch_one<BT, 3, false, T2>(p, num_sms, st, grid_out);
    if (red && p.n_acc == 1) return launch_one<BT, 1, true, T2>(p, num_sms, st, grid_out);
    if (red && p.n_acc == 2) return launch_one<BT, 2, true, T2>(p, num_sms, st, grid_out);
    if (red && p.n_acc == 3) return launch_one<BT, 3, true, T2>(p, num_sms, st, grid_out);
    return TBPM_EINVAL;
}

}  // namespace

// Instantiated: tiles of 1, 2, 4, 8 states; (n_acc, reduce) in {(0,0), (3,0), (1,1), (2,1), (3,1)}; WRITE_Y == !REDUCE.
bool term_ws_supported(int bt, const TermParams &p)
{
    if (p.n_table <= 0 || (p.flags & F_SKIP_H) || env_int("TBPM_DIRECT", 0)) return false;
    if (bt != 1 && bt != 2 && bt != 4 && bt != 8) return false;
    if ((int64_t)p.max_row_off * kConsumers > 12288) return false;               // index slice of a tile must fit a stage
    const bool red = p.flags & F_REDUCE, wy = p.flags & F_WRITE_Y;
    if (red == wy) return false;
    if (!red && !(p.n_acc == 0 || p.n_acc == 3)) return false;
    if (red && (p.n_acc < 1 || p.n_acc > 3)) return false;
    return true;
}

int launch_term_ws(int bt, TermParams p, int num_sms, cudaStream_t st, int *grid_out)
{
    const bool t2 = p.n_table == 1;
    switch (bt) {
    case 1: return t2 ? launch_variant<1, true>(p, num_sms, st, grid_out) : launch_variant<1, false>(p, num_sms, st, grid_out);
    case 2: return t2 ? launch_variant<2, true>(p, num_sms, st, grid_out) : launch_variant<2, false>(p, num_sms, st, grid_out);
    case 4: return t2 ? launch_variant<4, true>(p, num_sms, st, grid_out) : launch_variant<4, false>(p, num_sms, st, grid_out);
    case 8: return t2 ? launch_variant<8, true>(p, num_sms, st, grid_out) : launch_variant<8, false>(p, num_sms, st, grid_out);
    }
    return TBPM_EINVAL;
}

bool term_ph_supported(int bt, const TermParams &p)
{
    if (!term_ws_supported(bt, p)) return false;
    return p.max_row_off <= 8;                                                   // two stages of the widest tile fit 160 KB
}

}  // namespace tbpm_detail

// term.h -- private: parameters shared by the fused Chebyshev-term kernels (term_ws.cu, propagate.cu).
#pragma once

#include <cstdlib>
#include <unordered_map>

#include "tbpm_internal.h"

namespace tbpm_detail {

constexpr int kMaxBT = 32;       // widest state tile
constexpr int kMaxGrid = 4096;   // upper bound on the persistent grid (block partials are sized for it)

enum TermFlags { F_SUB_Y = 1, F_WRITE_Y = 2, F_SKIP_H = 4, F_ACC_INIT = 8, F_REDUCE = 16 };

// One launch = one Chebyshev term  T_k = a*H*T_{k-1} - T_{k-2}  on one tile of BT interleaved states
// (amxsy of PAPER.md:434/439), plus the deferred accumulation psi' += ca*T_k + cb*T_{k-1} + cc*T_{k-2}
// (the axpy of PAPER.md:440 for up to three terms at once) and, on the last term, <psi0|psi'> and <psi'|psi'>.
struct TermParams {
    // matrix: kernel layout (orp/ocol/oidx/vtab/diag) or canonical CSR (rowptr/col/val)
    const uint32_t *orp;
    const int32_t *ocol;
    const uint16_t *oidx;
    const double2 *vtab;
    const double *diag;
    const int64_t *rowptr;
    const int32_t *col;
    const double2 *val;
    int64_t n_orb;
    // vectors of this tile, [row][BT]
    const double2 *x;      // T_{k-1}
    double2 *y;            // T_{k-2} in, T_k out (in place)
    double2 *acc;          // psi'
    const double2 *psi0;   // bra of the correlation
    double *partial;       // [grid][BT][3]
    double a;              // 1/s (k = 1) or 2/s
    double2 ca, cb, cc;    // coefficients of T_k, T_{k-1}, T_{k-2} in this flush
    int n_acc;             // 0: psi' untouched; 1..3 terms added
    int flags;
    int n_table;           // entries of vtab (kernel layout)
    int max_row_off;       // longest off-diagonal row (sizes the staged index slices)
    int packed;            // n_table == 1: bit 31 of every ocol word = conjugate of the table value (build.cu)
    // warp-specialised kernel: shared-memory stage geometry (bytes), filled by its launcher
    int n_stage, stage_bytes, cap_entries, off_col, off_idx, off_diag, off_vec;
    int64_t walk_d0;       // phased kernel: tiles per lattice line (1: linear order)
    int walk_len;          // phased kernel: tiles per run of a block
    int64_t walk_stride;   // rows per lattice line (0: unknown)
    int walk_run;          // lines per run when walk_stride is used
    int n_lat_off;         // lattice strides found by the builder (uniform rows only), ascending
    int64_t lat_off[16];
    int64_t lat_delta[16]; // signed offsets of the sample row's entries, in slot order
    int pol;               // phased kernel: cache-policy bits (1: T_k stored evict-first)
    int reverse;           // phased kernel: sweep the tiles from the last row block to the first
    int uniform;           // every row holds exactly max_row_off off-diagonal entries
    int single_real;       // the table holds one value and it is real
};

// Two consecutive Chebyshev terms in ONE sweep (term_pair.cuh).  Phase 0 is term k (x = T_{k-1}, y = T_{k-2} -> T_k), phase 1 is
// term k+1 (x = T_k, y = T_{k-1} -> T_{k+1}); phase 1 of a tile runs a few hundred tiles behind phase 0, while T_k, T_{k-1} and the
// matrix slices are still in L2, so the pair moves matrix + 4 vectors through DRAM where two launches move 2 x (matrix + 3).
struct PhaseParams {
    const double2 *x;
    double2 *y;
    double a;
    double2 ca, cb, cc;
    int sub_y, n_acc, acc_init, reduce;
};

struct PairParams {
    TermParams t;          // matrix, n_orb, acc, psi0, partial, table / row-shape facts, stage geometry
    PhaseParams ph[2];
    int64_t halo;          // tiles: phase 1 of tile t needs phase 0 of every tile within +-halo (circular)
    int lag;               // steps of a block's sequence between phase 0 and phase 1 of its tiles
    int *progress;         // [grid] phase-0 tiles finished by each block (zeroed before the launch)
    int *error;            // set when a dependency wait gave up (never, unless the blocks are not co-resident)
};

// Table value of an entry: index in bits 0-14, bit 15 = take the conjugate (exact: only the sign bit of im changes).
__device__ __forceinline__ double2 table_value(double2 v, uint32_t idx)
{
    v.y = __longlong_as_double(__double_as_longlong(v.y) ^ ((long long)(idx >> 15) << 63));
    return v;
}

__device__ __forceinline__ void cfma(double2 &h, double2 v, double2 x)   // h += v * x (complex)
{
    h.x = fma(v.x, x.x, h.x);
    h.x = fma(-v.y, x.y, h.x);
    h.y = fma(v.x, x.y, h.y);
    h.y = fma(v.y, x.x, h.y);
}

// Experiment switches (TBPM_*): read from the environment once per tbpm_propagate / tbpm_ldos call -- env_epoch() is bumped
// at the start of every call -- not once per kernel launch.
inline unsigned long long &env_epoch()
{
    static thread_local unsigned long long e = 1;
    return e;
}
inline int env_int(const char *name, int dflt)
{
    struct Entry { unsigned long long epoch; int value; };
    static thread_local std::unordered_map<const char *, Entry> cache;   // keyed by the literal's address: one entry per call site
    Entry &c = cache[name];
    if (c.epoch != env_epoch()) {
        const char *e = std::getenv(name);
        c.value = e ? std::atoi(e) : dflt;
        c.epoch = env_epoch();
    }
    return c.value;
}

// Warp-specialised bulk-copy (TMA) kernel, term_ws.cu.  Returns TBPM_EINVAL if (bt, flags) has no instantiation
// (the caller then uses the direct kernel).  *grid_out = blocks launched (sizes the final reduction).
bool term_ws_supported(int bt, const TermParams &p);
int launch_term_ws(int bt, TermParams p, int num_sms, cudaStream_t st, int *grid_out);

// Phased kernel (term_ph.cuh): matrix slices staged by bulk copies, vectors streamed directly; one file per tile width.
bool term_ph_supported(int bt, const TermParams &p);
int launch_term_ph_bt1(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out);
int launch_term_ph_bt2(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out);
int launch_term_ph_bt4(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out);
int launch_term_ph_bt8(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out);

// Staged-gather kernel (term_sg.cu): tiles of 8 states on uniform lattices; false / TBPM_EINVAL when it does not apply.
bool term_sg_supported(int bt, const TermParams &p);
int launch_term_sg(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out);

// Pair kernel, one file per tile width (2, 4, 8 states).
int launch_term_pair_bt2(const PairParams &p, int num_sms, cudaStream_t st, int *grid_out);
int launch_term_pair_bt4(const PairParams &p, int num_sms, cudaStream_t st, int *grid_out);
int launch_term_pair_bt8(const PairParams &p, int num_sms, cudaStream_t st, int *grid_out);

}  // namespace tbpm_detail

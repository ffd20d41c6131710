// term.h -- private: parameters shared by the fused Chebyshev-term kernels (term_ph.cuh, propagate.cu).
#pragma once

#include "knobs.h"
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
    // two terms per sweep (term_sq2.cu): T_k -> out1, T_{k+1} = a2*H*T_k - T_{k-1} -> out2; ca, cb, cc, cd then belong to T_{k+1} .. T_{k-2}
    double2 *out1, *out2;
    double a2;
    double2 cd;
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
    const uint32_t *lat_flags;  // bit r: row r follows lat_delta exactly (build.cu, k_lat_flags)
    int64_t n_regular;     // number of such rows
    int64_t sq8_line;      // > 0: periodic square lattice with next-nearest neighbours whose hoppings depend on the in-line position
    int sq8_real_x;        // the hops along the line (directions 3, 4 of dline) are real
    const uint16_t *dline; // only (build.cu, k_sq8): line length in rows and the [x][8] table of value indices by direction
    const int16_t *d16;    // short rows, one real value (build.cu, k_near16): [row / 32][word][row % 32], +-1 flags | far offsets
    int n16_w;             // far offsets per row of d16 (1, 2 or 4), 0: none
    int lat_periodic3;     // the bits are those of the periodic three-dimensional lattice (wrapped neighbours count as regular)
    int pol;               // phased kernel: cache-policy bits (1: T_k stored evict-first)
    int reverse;           // phased kernel: sweep the tiles from the last row block to the first
    int uniform;           // every row holds exactly max_row_off off-diagonal entries
    int single_real;       // the table holds one value and it is real
    int device;            // CUDA device of the handle (per-device launch configuration caches)
    int zero;              // always 0, but known only at run time: the kernels AND it into the address of the barrier that hands a
                           // shared-memory stage back, together with the registers their LDS filled, so that the hand-back cannot be
                           // issued before those loads have returned
    int pf_dist;           // phased kernel: tiles ahead of the staged one whose vector rows are prefetched into L2 (0: off)
    int pf_mask;           // 1: y / psi' / psi0 rows, 2: x rows at the leading edge
    int64_t pf_lead;       // rows between a tile and the leading edge of its gather window (first touch of x)
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

// Shared-memory stage of the phased kernel: row offsets | column words | value indices | diagonal of one tile of R rows.
constexpr size_t kSmemMax = 227 * 1024;      // opt-in dynamic shared memory of one block on sm_100
constexpr size_t kStageBudget = 200 * 1024;  // what the stages of one block may take
constexpr int kMaxDevices = 64;
struct StageGeom { int cap_entries, off_col, off_idx, off_diag, stage_bytes; };
inline StageGeom stage_geom(int R, int max_row_off, bool with_idx)
{
    StageGeom g{};
    g.cap_entries = ((R * (max_row_off > 1 ? max_row_off : 1) + 8 + 7) / 8) * 8;   // + alignment slack of the slice start
    size_t o = (size_t)(((R + 1) * 4 + 15) & ~15);
    g.off_col = (int)o;  o += (size_t)g.cap_entries * 4;
    g.off_idx = (int)o;  o += with_idx ? (size_t)g.cap_entries * 2 : 0;
    o = (o + 15) & ~size_t(15);
    g.off_diag = (int)o; o += (size_t)((R * 8 + 15) & ~15);
    g.stage_bytes = (int)((o + 127) & ~size_t(127));
    return g;
}

// Phased kernel (term_ph.cuh): matrix slices staged by bulk copies, vectors streamed directly; one file per tile width.
// term_ph_supported: the tile width has an instantiation, the term is one of the five (n_acc, reduce) shapes, and two
// stages of the widest tile fit the shared memory of an SM (rows of up to a few dozen entries); everything else runs
// on the general kernel k_cheb_term (propagate.cu).
bool term_ph_supported(int bt, const TermParams &p);
int launch_term_ph_bt1(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out);
int launch_term_ph_bt2(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out);
int launch_term_ph_bt4(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out);
int launch_term_ph_bt8(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out);


// Rolling-window kernel (term_rw.cu): tiles of 8 states on lattices whose largest stride is a whole number of 128-row
// tiles; false / TBPM_EINVAL when it does not apply.
bool term_rw_supported(int bt, const TermParams &p);
int launch_term_rw(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out);

// Square-lattice kernel (term_sq.cu): tiles of 8 states on the periodic square lattice with next-nearest neighbours whose hopping
// values depend on the in-line position only; neither column words nor value indices are read per row.
bool term_sq_supported(int bt, const TermParams &p);
int launch_term_sq(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out);

// Two terms per sweep on the same lattice (term_sq2.cu); see launch_pair_sq for the meaning of the fields.
bool pair_sq_supported(int bt, const TermParams &p);
int launch_pair_sq(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out);

// Three-dimensional lattice kernel (term_l3.cu): tiles of 8 states on lattices with offsets {+-1, +-S1, +-S2} and one real hopping
// value (simple cubic and its anisotropic relatives); two-dimensional tiles with TMA-fed halos, walked along S2.
bool term_l3_supported(int bt, const TermParams &p);
int launch_term_l3(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out);


// Short-row kernel (term_n16.cu): tiles of ONE state (wider tiles stay on the phased kernel), rows of <= 4 entries no further than 32767 rows away, one real hopping
// value; reads the builder's 16-bit column offsets instead of row offsets and column words.
bool term_n16_supported(int bt, const TermParams &p);
int launch_term_n16(int bt, const TermParams &p, int num_sms, cudaStream_t st, int *grid_out);

}  // namespace tbpm_detail

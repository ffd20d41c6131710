// tbpm_internal.h -- private declarations of libtbpm.so (not part of the C ABI, not shared with oracle/).
#pragma once

#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include <atomic>
#include <mutex>
#include <vector>

#include "../../include/tbpm.h"

#define TBPM_CUDA_TRY(expr)                      \
    do {                                         \
        cudaError_t e__ = (expr);                \
        if (e__ != cudaSuccess) {                \
            tbpm_detail::note_cuda_error(e__);   \
            return TBPM_ECUDA;                   \
        }                                        \
    } while (0)

namespace tbpm_detail {

void note_cuda_error(cudaError_t e);
void count_launches(int n);   // process-wide kernel-launch counter (tbpm_total_launch_count)
long long total_launches();

constexpr size_t kAlign = 256;
inline size_t align_up(size_t v, size_t a = kAlign) { return (v + a - 1) / a * a; }

constexpr int kTableMax = 32768;        // distinct hopping values (v and conj v count once): 15-bit index + conjugate bit
constexpr int kHashSlots = 1 << 18;     // open-addressing table used while collecting distinct values
constexpr int kStatusWords = 64;

// status words written by the build kernels (device int32[kStatusWords] at the start of `persist`)
enum StatusWord {
    ST_ERR = 0,          // bit 0: index out of range, bit 1: diagonal hop, bit 2: duplicate (row, col)
    ST_MAX_ROW = 1,      // max entries in a row of the canonical CSR
    ST_GERSH_LO = 2,     // bits of the double max_i (|onsite_i| + sum_j |H_ij|)   (non-negative doubles order as u64)
    ST_GERSH_HI = 3,
    ST_NTAB = 4,         // number of distinct off-diagonal values inserted into the hash table
    ST_TAB_OVERFLOW = 5, // more than kTableMax distinct values (or a probe sequence gave up)
    ST_NEG_MIN_ROW = 6,  // 2^30 - (fewest entries in a row of the canonical CSR)
    ST_HALO = 7,         // widest |col - row| (circular): how far a row reaches into the vector
    ST_NREG = 8,         // rows whose entries sit exactly at the lattice offsets (k_lat_flags)
    ST_SQ8_BAD = 9,      // warps with a row that is not a site of the periodic square lattice with in-line hoppings (k_sq8)
    ST_N16_BAD = 10,     // warps with an entry further than 32767 rows from its row, also round the boundary (k_near16)
    ST_N16_WF = 11,      // most entries of a row that are not at row +- 1 (k_near16)
    ST_SQ8_CPLX = 12     // k_sq8: in-line hops (directions 3, 4) whose value has a non-zero imaginary part
};

// What the last tbpm_propagate / tbpm_ldos call of a handle left in a workspace (read by tbpm_get_state).
struct RunRecord {
    const void *workspace;
    int n_state, tile, last_bt;
    size_t vec0_off, full_vec;
};

}  // namespace tbpm_detail

// The handle: a host struct of device pointers into `persist`.
struct tbpm_ham {
    int64_t n_orb = 0;
    int64_t n_hop = 0;
    int64_t nnz = 0;       // canonical CSR entries
    int64_t nnz_off = 0;   // off-diagonal entries
    int has_onsite = 0;
    uint32_t flags = 0;
    int32_t max_row_nnz = 0;
    int32_t min_row_nnz = 0;
    int32_t single_real = 0;   // the table holds one value and it is real
    int32_t halo_rows = 0;     // widest circular |col - row|
    int32_t n_lat_off = 0;     // uniform rows: |col - row| of the entries of one sample row (lattice strides), ascending
    int64_t lat_off[16] = {0};
    int64_t lat_delta[16] = {0};   // the same offsets signed, in the order of the sample row's entries (slot j -> col - row)
    int64_t n_regular = 0;         // rows that follow lat_delta exactly (bits of lat_flags)
    int32_t sq8_real_x = 0;        // sq8_line > 0: the in-line hops (x direction) are all real (Landau gauge along the line)
    int64_t sq8_line = 0;          // > 0: periodic square lattice + next-nearest neighbours, line of this many rows, hoppings = dline
    int32_t near16_w = 0;          // > 0: d16 holds a flag word and this many far column offsets per row (term_n16.cu)
    int32_t lat_periodic3 = 0;     // the bits were computed for the periodic three-dimensional lattice (wrapped neighbours count)
    double gershgorin = 0.0;
    int32_t n_table = 0;   // 0: kernels read complex128 values from the canonical CSR
    int32_t packed = 0;    // n_table == 1: bit 31 of every ocol word = "conjugate of the table value" (oidx is not read by the kernels)
    int device = 0;
    int num_sms = 0;

    // canonical CSR (device)
    int64_t *rowptr = nullptr;
    int32_t *col = nullptr;
    double2 *val = nullptr;
    // kernel layout (device): off-diagonal part with 32-bit row offsets, 16-bit value indices and a real diagonal
    uint32_t *orp = nullptr;
    int32_t *ocol = nullptr;
    uint16_t *oidx = nullptr;
    double2 *vtab = nullptr;
    double *diag = nullptr;
    uint16_t *dline = nullptr;       // sq8_line > 0: value index of direction k at in-line position x, [x][8]
    int16_t *d16 = nullptr;          // near16_w > 0: [row / 32][word][row % 32], word 0 = +-1 flags, words 1.. = far col - row (modulo n_orb) of the row's entries in column order, 0 = no entry
    uint32_t *lat_flags = nullptr;   // uniform lattices: bit r = row r follows lat_delta exactly
    int32_t *status = nullptr;

    // options (tbpm_set_option)
    int opt_tile = 8;      // states per tile: 8 interleaved complex128 = one 128-byte line per row
    int opt_kernel = 0;    // 1: every term on the general kernel
    // bookkeeping of the propagate calls: written under `mu` (calls on distinct workspaces may run concurrently)
    mutable std::mutex mu;
    std::vector<tbpm_detail::RunRecord> runs;
    std::atomic<long long> last_launches{0};
};

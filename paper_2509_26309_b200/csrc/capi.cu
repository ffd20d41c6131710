// capi.cu -- the remaining C-ABI entry points: error strings and the end-to-end call on HOST buffers.
#include <atomic>
#include <cstdio>
#include <cstring>

#include "term.h"

using namespace tbpm_detail;

namespace {
thread_local char g_cuda_msg[256] = "CUDA runtime error";
std::atomic<long long> g_total_launches{0};
}

void tbpm_detail::note_cuda_error(cudaError_t e)
{
    std::snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA runtime error: %s (%s)", cudaGetErrorName(e), cudaGetErrorString(e));
}

void tbpm_detail::count_launches(int n) { g_total_launches.fetch_add(n, std::memory_order_relaxed); }
long long tbpm_detail::total_launches() { return g_total_launches.load(std::memory_order_relaxed); }

#ifdef TBPM_EXPERIMENT
// Experiment build only: a process-wide table of tuning knobs, set through tbpm_set_knob (not part of include/tbpm.h).
namespace {
struct KnobEntry { char name[32]; int value; };
KnobEntry g_knobs[64];
int g_n_knobs = 0;
}
int tbpm_detail::knob(const char *name, int dflt)
{
    for (int i = 0; i < g_n_knobs; ++i)
        if (std::strcmp(g_knobs[i].name, name) == 0) return g_knobs[i].value;
    return dflt;
}
extern "C" void tbpm_clear_knobs(void) { g_n_knobs = 0; }
extern "C" int tbpm_set_knob(const char *name, int value)
{
    if (!name || std::strlen(name) >= sizeof(g_knobs[0].name)) return TBPM_EINVAL;
    for (int i = 0; i < g_n_knobs; ++i)
        if (std::strcmp(g_knobs[i].name, name) == 0) { g_knobs[i].value = value; return TBPM_OK; }
    if (g_n_knobs >= 64) return TBPM_ENOMEM;
    std::strcpy(g_knobs[g_n_knobs].name, name);
    g_knobs[g_n_knobs++].value = value;
    return TBPM_OK;
}
#endif

// Does the phased kernel have an instantiation for this term whose stages fit one SM?  (see term.h)
bool tbpm_detail::term_ph_supported(int bt, const TermParams &p)
{
    if (p.n_table <= 0 || (p.flags & F_SKIP_H)) return false;
    if (bt != 1 && bt != 2 && bt != 4 && bt != 8) return false;
    const bool red = p.flags & F_REDUCE, wy = p.flags & F_WRITE_Y;
    if (red == wy) return false;
    if (!red && !(p.n_acc == 0 || p.n_acc == 3)) return false;
    if (red && (p.n_acc < 1 || p.n_acc > 3)) return false;
    const int lanes_per_row = bt >= 2 ? bt / 2 : 1;        // threads hold two states of a row (one at bt = 1)
    const int rows_max = 31 * 32 / lanes_per_row;          // the widest tile any shape of this width uses
    return 2 * (size_t)stage_geom(rows_max, p.max_row_off, true).stage_bytes <= kStageBudget;
}

extern "C" int64_t tbpm_total_launch_count(void) { return (int64_t)g_total_launches.load(std::memory_order_relaxed); }

extern "C" const char *tbpm_strerror(int code)
{
    switch (code) {
    case TBPM_OK: return "success";
    case TBPM_EINVAL: return "invalid argument (null, negative, misaligned, n_orb >= 2^31 or nnz >= 2^32 - 1)";
    case TBPM_EINDEX: return "hop or site index out of range";
    case TBPM_EDIAG: return "hop with i == j is illegal; on-site energies go into `onsite` (PAPER.md:177-179)";
    case TBPM_EDUP: return "duplicate (row, col) pair in the hopping list";
    case TBPM_ENOMEM: return "caller-provided buffer too small";
    case TBPM_ECUDA: return g_cuda_msg;
    case TBPM_EBOUND: return "Gershgorin bound of H exceeds rescale: the Chebyshev recursion would diverge";
    case TBPM_ETOOBIG: return "tbpm_propagate_static: the problem needs more workspace than the library's static array (TBPM_STATIC_WORKSPACE_BYTES)";
    }
    return "unknown error code";
}

extern "C" const char *tbpm_version(void)
{
#ifdef TBPM_EXPERIMENT
    return "tbpm-b200 0.2 (sm_100a) +exp";
#else
    return "tbpm-b200 0.2 (sm_100a)";
#endif
}

namespace {

struct Arena {
    size_t hop_i, hop_j, hop_val, onsite, psi0, corr, norm2, persist, scratch, workspace, total;
    size_t persist_bytes, scratch_bytes, workspace_bytes;
};

int arena_layout(int64_t n_orb, int64_t n_hop, int has_onsite, int n_state, int n_step, uint32_t flags, Arena *A)
{
    if (n_state < 0 || n_step < 0) return TBPM_EINVAL;
    int rc = tbpm_build_bytes(n_orb, n_hop, has_onsite, flags, &A->persist_bytes, &A->scratch_bytes);
    if (rc) return rc;
    tbpm_ham tmp;                                        // only n_orb (and the default options) matter for the workspace size
    tmp.n_orb = n_orb;
    if ((rc = tbpm_propagate_bytes(&tmp, n_state, &A->workspace_bytes))) return rc;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o += align_up(bytes ? bytes : 1); return at; };
    A->hop_i = take(sizeof(int32_t) * (size_t)n_hop);
    A->hop_j = take(sizeof(int32_t) * (size_t)n_hop);
    A->hop_val = take(sizeof(double) * 2 * (size_t)n_hop);
    A->onsite = take(has_onsite ? sizeof(double) * (size_t)n_orb : 0);
    A->psi0 = take(sizeof(double) * 2 * (size_t)n_orb * (size_t)n_state);
    A->corr = take(sizeof(double) * 2 * (size_t)n_state * (size_t)n_step);
    A->norm2 = take(sizeof(double) * (size_t)n_state * (size_t)n_step);
    A->persist = take(A->persist_bytes);
    A->scratch = take(A->scratch_bytes);
    A->workspace = take(A->workspace_bytes);
    A->total = o;
    return TBPM_OK;
}

}  // namespace

extern "C" int tbpm_corr_host_bytes(int64_t n_orb, int64_t n_hop, int has_onsite, int n_state, int n_step, uint32_t flags,
                                    size_t *arena_bytes)
{
    if (!arena_bytes) return TBPM_EINVAL;
    Arena A{};
    int rc = arena_layout(n_orb, n_hop, has_onsite, n_state, n_step, flags, &A);
    if (rc) return rc;
    *arena_bytes = A.total;
    return TBPM_OK;
}

extern "C" int tbpm_corr_host(int64_t n_orb, const double *onsite, int64_t n_hop, const int32_t *hop_i, const int32_t *hop_j,
                              const double *hop_val, uint32_t flags, const double *psi0, int n_state, int n_step, double dt,
                              double rescale, double *corr, double *norm2, void *arena, size_t arena_bytes, void *stream,
                              size_t *h2d_bytes, size_t *d2h_bytes)
{
    Arena A{};
    int rc = arena_layout(n_orb, n_hop, onsite != nullptr, n_state, n_step, flags, &A);
    if (rc) return rc;
    if (!arena || (reinterpret_cast<uintptr_t>(arena) & 255u)) return TBPM_EINVAL;
    if (arena_bytes < A.total) return TBPM_ENOMEM;
    if (n_hop > 0 && (!hop_i || !hop_j || !hop_val)) return TBPM_EINVAL;
    if (n_state > 0 && n_step > 0 && (!psi0 || !corr)) return TBPM_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    char *D = static_cast<char *>(arena);
    size_t up = 0, down = 0;
    auto h2d = [&](size_t off, const void *src, size_t bytes) -> int {
        if (bytes == 0) return TBPM_OK;
        TBPM_CUDA_TRY(cudaMemcpyAsync(D + off, src, bytes, cudaMemcpyHostToDevice, st));
        up += bytes;
        return TBPM_OK;
    };
    if ((rc = h2d(A.hop_i, hop_i, sizeof(int32_t) * (size_t)n_hop))) return rc;
    if ((rc = h2d(A.hop_j, hop_j, sizeof(int32_t) * (size_t)n_hop))) return rc;
    if ((rc = h2d(A.hop_val, hop_val, sizeof(double) * 2 * (size_t)n_hop))) return rc;
    if (onsite && (rc = h2d(A.onsite, onsite, sizeof(double) * (size_t)n_orb))) return rc;
    // psi0 goes up on a stream of its own, one tile of states at a time, so that the copy of tile t + 1 (and later) overlaps the
    // build and the propagation of the tiles before it; the tiles are independent, so the results are those of one call, bit for bit.
    const int tile = 8;
    const int n_tile = (n_state + tile - 1) / tile;
    cudaStream_t cs = nullptr;
    std::vector<cudaEvent_t> ev((size_t)std::max(n_tile, 0), nullptr);
    auto cleanup = [&]() {
        for (cudaEvent_t e : ev) if (e) cudaEventDestroy(e);
        if (cs) cudaStreamDestroy(cs);
    };
    if (n_state > 0 && n_step > 0 && n_orb > 0) {
        if (cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking) != cudaSuccess) { note_cuda_error(cudaGetLastError()); return TBPM_ECUDA; }
        cudaEvent_t e0 = nullptr;                           // whatever the caller queued on `stream` before this call comes first
        if (cudaEventCreateWithFlags(&e0, cudaEventDisableTiming) == cudaSuccess) {
            cudaEventRecord(e0, st);
            cudaStreamWaitEvent(cs, e0, 0);
            cudaEventDestroy(e0);
        }
        for (int t = 0; t < n_tile; ++t) {
            const int s0 = t * tile, ns = std::min(tile, n_state - s0);
            const size_t off = sizeof(double) * 2 * (size_t)n_orb * (size_t)s0, bytes = sizeof(double) * 2 * (size_t)n_orb * (size_t)ns;
            if (cudaEventCreateWithFlags(&ev[t], cudaEventDisableTiming) != cudaSuccess ||
                cudaMemcpyAsync(D + A.psi0 + off, reinterpret_cast<const char *>(psi0) + off, bytes, cudaMemcpyHostToDevice, cs) != cudaSuccess ||
                cudaEventRecord(ev[t], cs) != cudaSuccess) {
                note_cuda_error(cudaGetLastError());
                cudaStreamSynchronize(cs);
                cleanup();
                return TBPM_ECUDA;
            }
            up += bytes;
        }
    }

    tbpm_ham *H = nullptr;
    rc = tbpm_build(n_orb, onsite ? reinterpret_cast<const double *>(D + A.onsite) : nullptr, n_hop,
                    reinterpret_cast<const int32_t *>(D + A.hop_i), reinterpret_cast<const int32_t *>(D + A.hop_j),
                    reinterpret_cast<const double *>(D + A.hop_val), flags, D + A.persist, A.persist_bytes, D + A.scratch,
                    A.scratch_bytes, stream, &H);
    if (rc) { if (cs) cudaStreamSynchronize(cs); cleanup(); return rc; }
    if (H->opt_tile != tile) { tbpm_free(H); if (cs) cudaStreamSynchronize(cs); cleanup(); return TBPM_EINVAL; }
    for (int t = 0; t < n_tile && !rc && cs; ++t) {
        const int s0 = t * tile, ns = std::min(tile, n_state - s0);
        if (cudaStreamWaitEvent(st, ev[t], 0) != cudaSuccess) { note_cuda_error(cudaGetLastError()); rc = TBPM_ECUDA; break; }
        rc = tbpm_propagate(H, reinterpret_cast<const double *>(D + A.psi0) + 2 * (size_t)n_orb * (size_t)s0, ns, n_step, dt, rescale,
                            reinterpret_cast<double *>(D + A.corr) + 2 * (size_t)s0 * (size_t)n_step,
                            reinterpret_cast<double *>(D + A.norm2) + (size_t)s0 * (size_t)n_step, D + A.workspace, A.workspace_bytes, stream);
    }
    tbpm_free(H);
    if (rc) { if (cs) cudaStreamSynchronize(cs); cudaStreamSynchronize(st); cleanup(); return rc; }
    const size_t nc = (size_t)n_state * (size_t)n_step;
    if (nc > 0) {
        TBPM_CUDA_TRY(cudaMemcpyAsync(corr, D + A.corr, sizeof(double) * 2 * nc, cudaMemcpyDeviceToHost, st));
        down += sizeof(double) * 2 * nc;
        if (norm2) {
            TBPM_CUDA_TRY(cudaMemcpyAsync(norm2, D + A.norm2, sizeof(double) * nc, cudaMemcpyDeviceToHost, st));
            down += sizeof(double) * nc;
        }
    }
    const cudaError_t se = cudaStreamSynchronize(st);
    cleanup();
    TBPM_CUDA_TRY(se);
    if (h2d_bytes) *h2d_bytes = up;
    if (d2h_bytes) *d2h_bytes = down;
    return TBPM_OK;
}

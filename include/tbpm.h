/*
 * tbpm.h -- C ABI of libtbpm.so: the B200-native (sm_100a) hot path of TBPLaS 2.0's tight-binding propagation
 * method (TBPM), arxiv 2509.26309.  Citations are "PAPER.md:LINE" of the paper text plus the section.
 *
 * The path:
 *   a0  tbpm_build      hopping list (each conjugate pair once) -> canonical CSR on the device
 *                       (+ the internal compressed layout the kernels read)
 *   a1  coefficients    c_k = (2 - delta_k0)(-i)^k J_k(tau), truncated at |J_k| < 1e-15 ("the imaginary
 *                       factor ... has been merged into the Chebyshev coefficients"; values: BASELINE.json:configs[0])
 *   a2-a7 tbpm_propagate  per time step  psi <- sum_k c_k T_k(H/s) psi  by the recursion of PAPER.md:437-443
 *                       (p2 = p0; amxsy(2.0, p1, p0); axpy(coeff[n], p2, wf_out); rotate), then
 *                       corr[n] = <psi0|psi(t_n)> and norm2[n] = <psi|psi>   (calc_corr_dos)
 *   a8  tbpm_ldos       the same with psi0 = unit vectors on the given sites
 *
 * Conventions
 *   - "device" pointers are CUDA device memory of the current device; "host" pointers are ordinary host memory.
 *   - complex128 values are (re, im) pairs of doubles.  hbar = 1: dt is in 1/(energy unit of H); tau = rescale*dt.
 *   - Ownership: every buffer is allocated and freed by the caller (PyTorch in this repository).  The library
 *     allocates no device memory.  `persist` must outlive the handle; `scratch` may be released when tbpm_build
 *     returns; `workspace` holds the states of the last tbpm_propagate / tbpm_ldos call (see tbpm_get_state).
 *   - All device pointers must be 16-byte aligned; `persist`, `scratch`, `workspace` 256-byte aligned.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - Every function returns TBPM_OK (0) or a negative TBPM_E* code; no C++ exception crosses the ABI.
 *   - There is NO CPU fallback: without a usable CUDA device every device entry point returns TBPM_ECUDA.
 */
#ifndef TBPM_H
#define TBPM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tbpm_ham tbpm_ham; /* opaque host handle pointing into caller-owned device memory */

/* error codes */
#define TBPM_OK 0
#define TBPM_EINVAL (-1)  /* NULL / negative / misaligned argument, n_orb >= 2^31, rescale <= 0, ...                 */
#define TBPM_EINDEX (-2)  /* hop, site or state index out of range                                                    */
#define TBPM_EDIAG (-3)   /* hop with i == j: illegal, on-site energy is an orbital attribute    */
#define TBPM_EDUP (-4)    /* the same (row, col) produced twice (the paper's dict-update semantic, PAPER.md:190-191,
                             has no meaning for a flat list; SURVEY reading #15)                                     */
#define TBPM_ENOMEM (-5)  /* a caller-provided buffer is too small                                                   */
#define TBPM_ECUDA (-6)   /* CUDA runtime error (no device, launch failure, sticky error)                            */
#define TBPM_EBOUND (-7)  /* Gershgorin bound max_i(|onsite_i| + sum_j |H_ij|) > rescale (strictly): the Chebyshev
                             recursion would diverge.  Returned by tbpm_check_bound only; never fatal elsewhere.     */
#define TBPM_ETOOBIG (-8) /* tbpm_propagate_static: the problem needs more than TBPM_STATIC_WORKSPACE_BYTES of workspace       */

/* flags of tbpm_build */
#define TBPM_VALIDATE 1u    /* accepted and ignored: the precondition checks (index range, i != j, duplicates) ride on
                               kernels that run anyway and are reported through the status word that tbpm_build has to
                               read back for the table size, so they are ALWAYS on (the paper's "bugs vs exceptions"
                               split, would make them optional)                             */
#define TBPM_HOPS_FULL 2u   /* the list already holds both orientations of every pair (default: each pair once and
                               the conjugate partner H_ji = conj(H_ij) is generated)                    */
#define TBPM_NO_TABLE 4u    /* keep complex128 values in the kernel layout instead of 16-bit indices into a table of
                               distinct hopping values (the table is the default whenever <= 32768 values occur,
                               v and conj(v) counting once)                                                            */

const char *tbpm_strerror(int code);
const char *tbpm_version(void);

/* ---- a1: Chebyshev coefficients (host only, needs no GPU) -----------------------------------------------------------
 * tau >= 0.  K = first k >= ceil(tau) with |J_k(tau)| < tol (strict); coefficients k = 0..K-1 are written to
 * coeff[k][2].  K(pi) = 21 at tol = 1e-15, i.e. 20 H-applications per time step.  TBPM_ENOMEM if K > kcap (K is still
 * reported).  The library uses tol = 1e-15 (BASELINE.json:configs[0]). */
int tbpm_cheb_coeff(double tau, double tol, int kcap, int *K, double *coeff /* host [kcap][2] */);

/* ---- a0: build -----------------------------------------------------------------------------------------------------
 * Sizes of the two caller-provided device buffers for a model with n_orb orbitals and n_hop list entries. */
int tbpm_build_bytes(int64_t n_orb, int64_t n_hop, int has_onsite, uint32_t flags, size_t *persist_bytes,
                     size_t *scratch_bytes);

/* Entry h of the list means <hop_i[h]| H |hop_j[h]> = hop_val[h] (the paper's <i,0|H|j,R>); unless
 * TBPM_HOPS_FULL is set the partner <j|H|i> = conj(val) is added.  onsite (real, may be NULL) adds a diagonal entry
 * (onsite_i, 0) to EVERY row; onsite == NULL stores no diagonal.  Result: canonical CSR (rows ascending, columns
 * strictly ascending within a row), bit-exact whatever the order of the list, plus the internal kernel layout.
 * Rows without entries are legal.  The call enqueues its kernels on `stream` and synchronises it before returning
 * (it must read back the status word and the size of the hopping-value table). */
int tbpm_build(int64_t n_orb, const double *onsite /* device [n_orb] or NULL */, int64_t n_hop,
               const int32_t *hop_i /* device [n_hop] */, const int32_t *hop_j /* device [n_hop] */,
               const double *hop_val /* device [n_hop][2] */, uint32_t flags, void *persist /* device */,
               size_t persist_bytes, void *scratch /* device */, size_t scratch_bytes, void *stream, tbpm_ham **out);

/* nnz = stored entries of the canonical CSR; matrix_bytes_per_term = bytes of H the kernels read per Chebyshev term
 * (the "matrix bytes as stored" of the roofline count); n_table = distinct off-diagonal values (0: table not used);
 * gershgorin = max_i (|onsite_i| + sum_j |H_ij|).  Any output pointer may be NULL. */
int tbpm_ham_info(const tbpm_ham *H, int64_t *n_orb, int64_t *nnz, int32_t *max_row_nnz, size_t *matrix_bytes_per_term,
                  int32_t *n_table, double *gershgorin);

/* Lattices the builder recognises: tiles of 8 states then run on a kernel that reads no column words and
 * no per-entry value indices for the rows that sit on the lattice.  kind: 0 none, TBPM_LATTICE_CUBIC (offsets {+-1, +-S1, +-S2},
 * one real hopping value: BASELINE.json:configs[4]), TBPM_LATTICE_SQUARE8 (periodic square lattice with next-nearest neighbours,
 * hoppings that depend on the in-line position only: configs[3]); and, for tiles of ONE state, TBPM_LATTICE_NEAR16 (rows of
 * at most 4 off-diagonal entries, none further than 32767 rows from its own, one real hopping value -- honeycomb or square lattice
 * with vacancies or on-site disorder: configs[0..2]; that kernel reads 16-bit column offsets).  bytes_per_term = the bytes of H THAT
 * kernel reads per Chebyshev term (what bench.py counts as the matrix when it runs on it); 0 when kind is 0.  Outputs may be NULL. */
#define TBPM_LATTICE_CUBIC 2
#define TBPM_LATTICE_SQUARE8 3
#define TBPM_LATTICE_NEAR16 4
int tbpm_ham_lattice_info(const tbpm_ham *H, int32_t *kind, size_t *bytes_per_term);

/* TBPM_EBOUND if gershgorin > rescale (test is '>' : config 4 sits exactly at equality), else TBPM_OK. */
int tbpm_check_bound(const tbpm_ham *H, double rescale);

/* Canonical CSR in caller order, copied device -> device: rowptr int64[n_orb+1], col int32[nnz], val [nnz][2]. */
int tbpm_export_csr(const tbpm_ham *H, int64_t *rowptr, int32_t *col, double *val, void *stream);

/* Frees only the host struct (PAPER.md has no counterpart: its solver holds `const model_t*`).  Work
 * enqueued on the handle must have completed. */
void tbpm_free(tbpm_ham *H);

/* Options of a handle; set before tbpm_propagate_bytes / tbpm_propagate / tbpm_ldos (the workspace size depends on
 * TBPM_OPT_TILE).  The library reads nothing from the environment: its behaviour is a function of its arguments. */
#define TBPM_OPT_TILE 1   /* states propagated together per tile (SpMM width, PAPER.md:554 runs one state at a time):
                             1, 2, 4, 8 (default: 8 interleaved complex128 = one 128-byte line per row), 16, 32        */
#define TBPM_OPT_KERNEL 2 /* 0 (default): the fastest kernel that applies (tiles of 8 states on a recognised lattice: the
                             three-dimensional / square-lattice / rolling-window kernel; tiles of one state on short rows with one
                             real value: the 16-bit-offset kernel; else phased; else general);
                             1: every term on the general kernel; 2: no lattice kernel (phased, else general);
                             3: of the lattice kernels only the rolling-window one (tests); 4: as 0, but always ONE Chebyshev
                             term per launch (0 runs two terms per sweep on the square lattice of configs[3], which needs two
                             more vectors of workspace: tbpm_propagate_bytes accounts for them)                          */
int tbpm_set_option(tbpm_ham *H, int option, int64_t value);

/* ---- a2-a7: propagate ------------------------------------------------------------------------------------------------
 * Size of the caller-owned `workspace` for n_state states: four vectors [n_orb][tile] complex128 per tile of states (the
 * rotating p0 / p1 / wf_out of PAPER.md:437-443 and the bra psi0 of calc_corr_dos) + block partials, + two more
 * vectors of one tile where the two-terms-per-sweep kernel applies (a smaller workspace of at least the plain size is accepted:
 * the call then runs one term per sweep). */
int tbpm_propagate_bytes(const tbpm_ham *H, int n_state, size_t *workspace_bytes);

/* psi0: device [n_state][n_orb][2], state-major (one random initial state per row; one independent propagation per
 * state).  corr: device out [n_state][n_step][2], entry n is t = (n+1)*dt (t = 0, value <psi0|psi0>, is
 * not stored).  norm2: device out [n_state][n_step] or NULL.  rescale = s > 0 must bound the spectrum, ||H|| <= s
 * (config.rescale).  n_step == 0 or n_state == 0: success, outputs untouched.  Asynchronous on `stream`.
 * Deterministic: the same inputs give bit-identical outputs, and the first m entries do not depend on n_step. */
int tbpm_propagate(tbpm_ham *H, const double *psi0, int n_state, int n_step, double dt, double rescale,
                   double *corr, double *norm2, void *workspace, size_t workspace_bytes, void *stream);

/* The same propagation for callers that CANNOT allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): no workspace argument -- the workspace is a file-scope device array of
 * TBPM_STATIC_WORKSPACE_BYTES inside the library (8 MiB, held by every GPU that loads the library until the process exits), and the
 * call performs no cudaMalloc / cudaFree / allocating library routine.  Inputs and outputs are the caller's, as in tbpm_propagate, and
 * the results are bit-identical to tbpm_propagate's.  Limits: tbpm_propagate_bytes(H, n_state) <= TBPM_STATIC_WORKSPACE_BYTES, i.e.
 * about n_orb x min(n_state, tile) <= 80,000 per tile (BASELINE.json:configs[0] with up to 8 states), else TBPM_ETOOBIG and nothing
 * is launched; the handle's device must be the current device (TBPM_EINVAL).  The array is shared by every call on that device and
 * keeps the last call's contents (each call initialises what it reads); calls that OVERLAP on the GPU -- two streams, two host
 * threads -- race on it: serialise them.  tbpm_get_state does not apply to this call's workspace.  The first call on a device looks
 * the array's address up (cudaGetSymbolAddress): make that call outside a graph capture. */
#define TBPM_STATIC_WORKSPACE_BYTES (8u << 20)
int tbpm_propagate_static(tbpm_ham *H, const double *psi0, int n_state, int n_step, double dt, double rescale,
                          double *corr, double *norm2, void *stream);

/* ---- a8: TBPM-style LDOS correlation: psi0_b = e_{sites[b]}, corr[b][n] = <site_b| psi_b(t_n) > ----------------------
 * BASELINE.json:configs[4] ("LDOS correlation on 64 seeded site-localized initial states"); the paper's own LDOS is the
 * Haydock recursion, see tbpm_haydock below.  Same kernels as tbpm_propagate with unit initial vectors. */
int tbpm_ldos(tbpm_ham *H, const int64_t *sites /* host [n_site] */, int n_site, int n_step, double dt,
              double rescale, double *corr, double *norm2, void *workspace, size_t workspace_bytes, void *stream);

/* State `state` as left in `workspace` by the last tbpm_propagate / tbpm_ldos call of THIS handle on it (psi after its
 * n_step steps), caller order, device out [n_orb][2].  A snapshot at step j is a call with n_step = j: this is the
 * time-dependent wave function psi(t_j) the paper's solver can dump (WFT, Table 7), and
 * what the windowed parity protocol of SURVEY.md 8(d)(3) downloads.  TBPM_EINVAL if the handle has not propagated on
 * that workspace, TBPM_EINDEX if state >= the n_state of that call. */
int tbpm_get_state(const tbpm_ham *H, const void *workspace, int state, double *psi_out, void *stream);

/* Number of kernels the last tbpm_propagate / tbpm_ldos call on this handle launched (host counter kept in the handle). */
int64_t tbpm_last_launch_count(const tbpm_ham *H);
/* Kernels launched by this library in this process since it was loaded (build + propagate + get_state). */
int64_t tbpm_total_launch_count(void);

/* ---- NEXT-1: DOS from the correlation function (`Analyzer.calc_dos(corr)`) ----------------
 * The paper prints no formula; reading #27: average corr over the states, C_0 = 1, C_{-n} = conj(C_n), Hann window
 * w_n = (1 + cos(pi n / n_step)) / 2, and
 *     dos[j] = (dt / 2 pi) * [ 1 + 2 Re sum_{n=1}^{n_step} w_n C_n exp(+i n E_j dt) ],   E_j = -rescale + j * rescale / n_step,
 * j = 0 .. 2 n_step (at dt = pi / rescale the sampling interval matches the window [-rescale, rescale] and the sum of dos[j]
 * times the grid step is 1).  corr: device [n_state][n_step][2] as written by tbpm_propagate / tbpm_ldos; energy, dos: device
 * out [2 n_step + 1].  Plain direct transform (n_step <= a few thousand), one thread per energy.  Asynchronous on `stream`. */
int tbpm_dos(const double *corr, int n_state, int n_step, double dt, double rescale, double *energy, double *dos, void *stream);

/* ---- NEXT-3: quasi-eigenstates (QE) and the time-dependent wave function (WFT) ----------------------------------------------
 * "quasi-eigenstates (QE) and time-dependent wave function (WFT)" are solver functions of the paper (Table 7,
 * PAPER.md:1748-1749); it prints no formula (the TBPM mathematics is deferred to the v1.3 article).
 * reading #28: the one-sided, Hann-windowed Fourier transform of psi(t) at the requested energies, NOT normalised,
 *     qe[b][e] = sum_{n=0}^{n_step} w_n exp(+i E_e n dt) psi_b(n dt),   w_n = (1 + cos(pi n / n_step)) / 2,   psi_b(0) = psi0[b],
 * accumulated during the same propagation that yields corr / norm2 (same arguments and results as tbpm_propagate).  WFT is
 * tbpm_get_state after a call with n_step = j.  energies: host [n_energy], n_energy <= 16, in the energy unit of H.
 * qe: device out [n_state][n_energy][n_orb][2].  The workspace is that of tbpm_propagate plus n_energy vectors of one tile. */
int tbpm_propagate_qe_bytes(const tbpm_ham *H, int n_state, int n_energy, size_t *workspace_bytes);
int tbpm_propagate_qe(tbpm_ham *H, const double *psi0, int n_state, int n_step, double dt, double rescale,
                      const double *energies /* host */, int n_energy, double *corr, double *norm2, double *qe /* device out */,
                      void *workspace, size_t workspace_bytes, void *stream);

/* ---- NEXT-2: Haydock recursion ("LDOS using Haydock recursive method"; Table 7) ----
 * The paper prints no formula; reading #29, the textbook recursion from |phi_0> = |site>:
 *     a_n = <phi_n|H|phi_n>,   b_{n+1} phi_{n+1} = H phi_n - a_n phi_n - b_n phi_{n-1},   b_{n+1} = || . ||,   b_0 phi_{-1} = 0.
 * a: device out [n_site][n_iter] = a_0 .. a_{n_iter-1};  b: device out [n_site][n_iter] = b_1 .. b_{n_iter}.  The LDOS follows on
 * the host from the continued fraction G(z) = 1 / (z - a_0 - b_1^2 / (z - a_1 - ...)) (kilobytes; see oracle.haydock_ldos).
 * H is NOT rescaled.  After a breakdown (b = 0: Krylov space exhausted) the remaining coefficients are 0.  sites: host [n_site].
 * workspace: tbpm_propagate_bytes(H, n_site).  Two sweeps per iteration: H u_n fused with <u_n|H u_n> (the fused last-term
 * kernel), then the three-vector update fused with the norm. */
int tbpm_haydock(tbpm_ham *H, const int64_t *sites /* host */, int n_site, int n_iter, double *a /* device out */,
                 double *b /* device out */, void *workspace, size_t workspace_bytes, void *stream);
/* The continued fraction on the device: ldos[s][j] = -Im G_s(energy[j] + i eta) / pi, cut after a_{n_iter-1} (the chain is simply
 * finite; b_{n_iter} is not used).  a, b: device [n_site][n_iter] as written by tbpm_haydock; energy: device [n_energy];
 * ldos: device out [n_site][n_energy]; eta > 0. */
int tbpm_haydock_ldos(const double *a, const double *b, int n_site, int n_iter, const double *energy, int n_energy, double eta,
                      double *ldos, void *stream);

/* ---- NEXT-4: AC-conductivity correlation function ("AC conductivity (AC)"; Table 7; the current
 * operator acts through a sparse matrix-vector product, and has a CSR of its own) ------------------
 * The paper prints no formula; reading #30 (hbar = e = 1):
 *     psi1(0) = [1 - f(H)] J_b psi0,   psi2(0) = f(H) psi0,   f(E) = 1 / (exp(beta (E - mu)) + 1),   psi_i(t) = exp(-i H t) psi_i(0),
 *     corr[b][n] = < psi2(n dt) | J_a | psi1(n dt) >,   n = 0 .. n_step      (device out [n_state][n_step + 1][2]).
 * Ja, Jb: handles built with tbpm_build from the hop lists of the current operators J = i [H, r] (entry <i|J|j> = i <i|H|j>
 * (r_i - r_j), Hermitian, so each conjugate pair once; no onsite), same n_orb and device as H.  f(H) and 1 - f(H) are applied by
 * their Chebyshev series on [-rescale, rescale] (tbpm_fermi_coeff: host only, real coefficients as (re, 0) pairs, truncated after
 * the last |c_k| >= tol; the library uses tol = 1e-13).  Workspace: tbpm_corr_ac_bytes (six vectors of one tile, + two where the two-terms-per-
 * sweep kernel applies; with only the six the series run one term per sweep). */
int tbpm_fermi_coeff(double beta, double mu, double rescale, int one_minus, double tol, int kcap, int *K, double *coeff /* host [kcap][2] */);
int tbpm_corr_ac_bytes(const tbpm_ham *H, int n_state, size_t *workspace_bytes);
int tbpm_corr_ac(tbpm_ham *H, tbpm_ham *Ja, tbpm_ham *Jb, const double *psi0 /* device [n_state][n_orb][2] */, int n_state, int n_step,
                 double dt, double rescale, double beta, double mu, double *corr /* device out */, void *workspace,
                 size_t workspace_bytes, void *stream);

/* Dynamic-polarisation correlation ("dynamic polarizability (DP)"; Table 7; no formula printed).
 * DESIGN.md reading #31: the scheme of tbpm_corr_ac with DIAGONAL density operators rho(q) = diag(exp(i q.r_i)) in place of the
 * current operators: psi1(0) = [1 - f(H)] (rho_b * psi0), psi2(0) = f(H) psi0, corr[b][n] = <psi2(n dt)| rho_a * psi1(n dt)>,
 * n = 0 .. n_step.  rho_a, rho_b: device [n_orb][2] (the caller passes rho_b = rho(-q), rho_a = rho(q)).  Workspace and output
 * as for tbpm_corr_ac. */
int tbpm_corr_dp(tbpm_ham *H, const double *rho_a /* device */, const double *rho_b /* device */, const double *psi0 /* device */, int n_state,
                 int n_step, double dt, double rescale, double beta, double mu, double *corr /* device out */, void *workspace,
                 size_t workspace_bytes, void *stream);

/* ---- end to end with HOST buffers ------------------------------------------------------------------------------------
 * Whole path for host-resident inputs: H2D of the list and psi0, tbpm_build, tbpm_propagate, D2H of corr/norm2, then a
 * stream synchronise.  `arena` is caller-owned device memory of at least tbpm_corr_host_bytes(); host buffers should be
 * pinned for full copy bandwidth.  h2d_bytes / d2h_bytes (may be NULL) report what was copied.  The arena is sized before the
 * lattice is known and holds the plain workspace only: on the square lattice of configs[3] this call therefore runs one Chebyshev
 * term per sweep (same results; use tbpm_build + tbpm_propagate for the two-terms-per-sweep kernel). */
int tbpm_corr_host_bytes(int64_t n_orb, int64_t n_hop, int has_onsite, int n_state, int n_step, uint32_t flags,
                         size_t *arena_bytes);
int tbpm_corr_host(int64_t n_orb, const double *onsite /* host or NULL */, int64_t n_hop, const int32_t *hop_i /* host */,
                   const int32_t *hop_j /* host */, const double *hop_val /* host */, uint32_t flags,
                   const double *psi0 /* host [n_state][n_orb][2] */, int n_state, int n_step, double dt, double rescale,
                   double *corr /* host out */, double *norm2 /* host out or NULL */, void *arena /* device */,
                   size_t arena_bytes, void *stream, size_t *h2d_bytes, size_t *d2h_bytes);

#ifdef __cplusplus
}
#endif
#endif /* TBPM_H */

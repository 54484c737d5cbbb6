/*
 * polfed.h -- C ABI of libpolfed: the POLFED hot path on one NVIDIA B200 (sm_100a).
 *
 * POLFED = polynomially filtered exact diagonalisation (arxiv/paper_2605_10191).  Citations
 * "PAPER.md:<line>" refer to the paper text this library was written from; "R<n>" to the
 * readings listed in DESIGN.md.
 *
 * Conventions
 *   - Every function returns an int status (POLFED_OK == 0).  polfed_last_error() returns a
 *     thread-local, NUL-terminated description of the last failure on the calling thread.
 *     No exception crosses this boundary.
 *   - Pointers prefixed d_ are DEVICE pointers (cudaMalloc / torch CUDA tensor data_ptr()),
 *     h_ are HOST pointers.  Scalars are passed by value.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Unless
 *     a function says it synchronises, work is only enqueued on that stream.
 *   - Vector blocks are N x s, row-major ("row-interleaved": the s entries of row i are
 *     contiguous, leading dimension s), fp64, 16-byte aligned.  s in {1,2,4,8,16,32}.
 *   - Opaque handles (polfed_basis, polfed_ham) are owned by the library and released by
 *     the matching *_destroy.  All blocks, outputs and workspaces are owned by the caller.
 *   - Basis states are unsigned integers; bit i is site i (0-based); bit value 1 = spin up
 *     (S^z = +1/2) = occupied (R12, R13).  States are ordered as ascending integers, so
 *     rank(x) = sum_{j=1..k} C(p_j, j) with p_1 < ... < p_k the set bits of x (combinatorial
 *     number system).  The full space (n_up < 0) has rank(x) = x.
 *   - Random numbers never cross this boundary: model parameters arrive as arrays.
 */
#ifndef POLFED_H
#define POLFED_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  POLFED_OK = 0,
  POLFED_EINVAL = 1,     /* bad argument (NULL, unsupported s, misaligned pointer, ...) */
  POLFED_ENOMEM = 2,     /* host or device allocation failed */
  POLFED_ECUDA = 3,      /* a CUDA call or kernel launch failed */
  POLFED_ERANGE = 4,     /* rescaled target outside (-1,1), b <= 0, index overflow */
  POLFED_ENOCONV = 5,    /* eigen-solver hit max_krylov_dim before nev pairs converged */
  POLFED_EBREAKDOWN = 6, /* rank-deficient Krylov block (R17) */
  POLFED_EWINDOW = 7     /* eigen-solver: every extracted pair converged, but the filter's main lobe
                            holds fewer than nev levels (order K too high); outputs are valid eigenpairs */
};

typedef struct polfed_basis polfed_basis;
typedef struct polfed_ham polfed_ham;

const char* polfed_last_error(void);
/* major*10000 + minor*100 + patch */
int polfed_version(void);
/* Returns the unused memory of the library's stream-ordered scratch pool on the current device
 * to the driver (polfed_filter_apply_host and the eigen-solver keep their scratch blocks in that
 * pool between calls, up to 6 blocks of n*s doubles, so that later calls do not allocate).
 * Synchronises the device.  Safe to call at any time; the next call allocates again. */
int polfed_release_scratch(void);

/* ------------------------------------------------------------------------------------------
 * Basis (the paper uses symmetry sectors but never says how they are
 * enumerated, PAPER.md:510-515, 962 -- R12).
 * ------------------------------------------------------------------------------------------ */

/* Enumerate on the device all x in [0, 2^n_sites) with popcount n_up, ascending
 * (n_up < 0: the full 2^n_sites space, no table is stored).  1 <= n_sites <= 62 and the
 * dimension must be < 2^31.  Synchronises `stream` before returning. */
int polfed_build_basis(int n_sites, int n_up, void* stream, polfed_basis** out);
int polfed_basis_destroy(polfed_basis* basis);
int polfed_basis_dim(const polfed_basis* basis, int64_t* dim);
/* Device pointer to the dim ascending states (library-owned, valid until destroy).  For the
 * full space the table is materialised on first call. */
int polfed_basis_states(const polfed_basis* basis, const uint64_t** d_states);
/* d_rank[t] = position of d_states[t] in the basis, or -1 if its popcount is not n_up or it
 * has a bit at or above n_sites.  n >= 0 entries; enqueued on `stream`. */
int polfed_basis_rank(const polfed_basis* basis, const uint64_t* d_states, int64_t n,
                      int64_t* d_rank, void* stream);

/* ------------------------------------------------------------------------------------------
 * Hamiltonian assembly.  One term list covers the paper's models: XXZ chain Eq. (54)
 * PAPER.md:858-863; quantum sun Eq. (67); the spinless-fermion chain of
 * BASELINE.json config 5 (R15).
 * ------------------------------------------------------------------------------------------ */
enum {
  POLFED_TERM_ZZ = 0,    /* amp * S^z_i S^z_j                     diagonal            */
  POLFED_TERM_Z = 1,     /* amp * S^z_i                           diagonal, j ignored */
  POLFED_TERM_NN = 2,    /* amp * n_i n_j                         diagonal            */
  POLFED_TERM_N = 3,     /* amp * n_i                             diagonal, j ignored */
  POLFED_TERM_EXCH = 4,  /* amp * (S^+_i S^-_j + h.c.)            XXZ: amp = J/2 (R13) */
  POLFED_TERM_HOPJW = 5, /* amp * (c^+_i c_j + h.c.) with Jordan-Wigner sign
                            (-1)^{# occupied sites strictly between i and j}           */
  POLFED_TERM_XX = 6     /* amp * 4 S^x_i S^x_j: flips bits i and j with amplitude amp */
};
typedef struct {
  int32_t i, j;
  double amp;
  int32_t kind;
} polfed_term;

/* Dense symmetric block acting on bits 0..n_bits-1 (the quantum-sun dot):
 * h_dense is a HOST array, 2^n_bits x 2^n_bits row-major.  Only valid on a full-space basis. */
typedef struct {
  int32_t n_bits;
  const double* h_dense;
} polfed_dense_block;

enum {
  POLFED_FORMAT_CSR = 0,
  /* 1 was SELL-8-sigma in round 1: slower than the CSR kernel on every config, removed */
  POLFED_FORMAT_TILED = 2, /* CSR plus the tiled structured format below */
  POLFED_FORMAT_FLIP = 3,  /* CSR plus the matrix-free flip format below */
  POLFED_FORMAT_SECTOR = 4 /* the tiled format with register-resident tile-local hops, below */
};

/* Assemble H on the device as CSR: row_ptr int32[N+1], col int32[nnz] ascending within a
 * row, val fp64[nnz].  The diagonal entry of every row is stored even when zero; entries
 * that fall on the same (row, col) are summed in term order (dot block first); the diagonal
 * is the sum of the dot-block diagonal and the diagonal terms in term order, each product
 * and sum rounded separately (no FMA), so values are reproducible bit for bit.
 * h_terms is a HOST array.  A term that leaves the basis gives POLFED_EINVAL.
 * Synchronises `stream` before returning. */
int polfed_build_hamiltonian(const polfed_basis* basis, const polfed_term* h_terms, int n_terms,
                             const polfed_dense_block* dot /* may be NULL */, int format,
                             void* stream, polfed_ham** out);
/* POLFED_FORMAT_TILED (the paper's "optimized mapping" for constant off-diagonal values,
 * PAPER.md:625-651, 779; north_star's structured alternative): besides the CSR, the handle gets
 * a tile table for chains whose hops conserve the particle number.  Rows that share their top
 * n_sites - m bits (m = ceil(n_sites/2)) are one tile; hops among the low m sites stay inside it
 * and are stored once per particle-number class as neighbour index + sign, grouped by the at
 * most 4 distinct |amp| values; hops among the high sites are tile-local in the site-reversed
 * row order; the diagonal and the few hops across the cut are kept per row (at most 7 such hops
 * per state, at most 15 distinct |amp| among them; one packed 32-bit word each).
 * polfed_filter_apply then runs the recurrence as sweeps that alternate between the two row
 * orders with the tile held in shared memory (same result up to rounding order).
 * Requirements (else POLFED_EINVAL): fixed-n_up basis of fewer than 2^26 states,
 * 4 <= n_sites <= 26, no dense block,
 * off-diagonal terms of kind EXCH or HOPJW only, at most 4 distinct |amp| and 24 hops per state
 * inside a tile.  Used by polfed_filter_apply for s in {16, 32}; every other entry point uses
 * the CSR.  On this path d_V and d_W must be 32-byte and d_work 128-byte aligned (POLFED_EINVAL
 * otherwise).  All mutable state of a filter application (tile counters included) lives in the
 * caller's d_work, so one handle may serve several streams at once with distinct workspaces.
 *
 * POLFED_FORMAT_SECTOR: the same two-layout pipeline for chains whose tile-local hops are one
 * amplitude on every bond (i, i+1) and none or one amplitude on every bond (i, i+2) (EXCH, or
 * HOPJW with its Jordan-Wigner sign), e.g. config 5 (t, t') and the XXZ chains (J/2).  The m tile
 * sites are split into two groups; a lane group holds all rows that differ only inside one group
 * (at most C(7,3) = 35) in registers and applies that group's hops as a compile-time operator, so
 * shared memory is touched about 5 times per row and phase instead of once per stored entry; only
 * the bonds between the groups and across the tile cut remain per-row gathers.  Blocks are
 * streamed as 8-column panels (64-byte rows), the tile twice in shared memory.  Requirements
 * beyond POLFED_FORMAT_TILED's (else POLFED_EINVAL): the bond pattern above in both row orders,
 * at most 3 hopping terms across the cut, ceil(n_sites/2) in {4..9, 13} (chains with (i, i+2)
 * bonds) or {6, 7, 8, 10} (without).  Same alignment rules and workspace ownership. */

/* POLFED_FORMAT_FLIP (matrix-free rows for full-space spin models, the paper's Fig. 7 kernel
 * `newstate = state XOR mask`; the quantum sun Eq. 67): besides the CSR, the
 * handle keeps the diagonal, the dense block embedded in an 8 x 8 matrix on bits 0-2 and one
 * (mask, amplitude) pair per XX term.  Every fused step on the handle with s in {8, 16, 32}
 * (polfed_fused_step, polfed_filter_apply, the eigen-solver, KPM) then generates the rows from
 * the masks: eight consecutive rows are held in registers, the dense part is applied there and
 * each XX term reads the eight rows of one partner block; same result up to rounding order.
 * Requirements (else POLFED_EINVAL): full space (n_up < 0), 3 <= n_sites <= 31, dense block on
 * at most 3 bits, off-diagonal terms of kind XX only, at most 64 of them outside bits 0-2. */

/* Wrap a caller-owned device CSR (any real symmetric matrix, columns < n, row_ptr[n] == nnz).
 * The three arrays are kept by pointer and must outlive the handle.  They must be COMPLETE when the
 * call is made: it launches kernels that read them (the longest row for n <= 262144; a scan of the
 * values) and synchronises before returning.  polfed_ham_from_csr runs that work on the legacy
 * default stream; use polfed_ham_from_csr_ex to give the stream the arrays were produced on.
 *
 * The VALUES ARE SNAPSHOTTED when the off-diagonal entries take one or two distinct values (every
 * XXZ chain): the handle then also holds a packed copy (dense diagonal + 4-byte column words,
 * 4 B per entry + 12 n bytes of device memory) and the fused-step kernel reads that copy, not
 * d_val (the persistent small-matrix filter still reads d_val).  A caller that later changes d_val
 * in place must either build a new handle or pass POLFED_HAM_NO_SNAPSHOT: the handle then holds no
 * copy of any value, skips that pass over the entries, and every step reads d_val as it is at that
 * moment (plain CSR kernel: 12 instead of 4 bytes per stored entry; XXZ L = 20, s = 16 in round 1:
 * 32.7 against 26.6 us per step).  The structure (row_ptr, col) must never change under a handle.
 * Errors: POLFED_EINVAL (NULL, negative size, d_val not 16-byte / d_col not 4-byte aligned, unknown
 * flag), POLFED_ERANGE (n or nnz >= 2^31), POLFED_ENOMEM, POLFED_ECUDA. */
enum { POLFED_HAM_NO_SNAPSHOT = 1 };
int polfed_ham_from_csr(int64_t n, int64_t nnz, const int32_t* d_row_ptr, const int32_t* d_col,
                        const double* d_val, polfed_ham** out);
int polfed_ham_from_csr_ex(int64_t n, int64_t nnz, const int32_t* d_row_ptr, const int32_t* d_col,
                           const double* d_val, unsigned flags, void* stream, polfed_ham** out);
int polfed_ham_destroy(polfed_ham* ham);
/* Any output pointer may be NULL. */
int polfed_ham_csr(const polfed_ham* ham, int64_t* n, int64_t* nnz, const int32_t** d_row_ptr,
                   const int32_t** d_col, const double** d_val);

/* ------------------------------------------------------------------------------------------
 * The hot path.
 * ------------------------------------------------------------------------------------------ */

/* One fused pass, the mapping f!(Y, X) of PAPER.md:657-659 merged with the three-term update
 * of Eq. (51) PAPER.md:427-431 and the rescaling of Eq. (31) PAPER.md:274-276:
 *
 *     Y[i,:] = p * sum_j H_ij X[j,:] + q * X[i,:] + r * Z[i,:] + c * V[i,:]
 *
 * d_Z is not read when r == 0 (may be NULL), d_V is not read when c == 0 (may be NULL).
 * d_Y may alias d_Z or d_V (row i of Z and V is read only by the threads that write row i
 * of Y); d_Y must not overlap d_X.  Also serves H X (p=1), Eq. (28)-(30) (KPM recurrence)
 * and the Lanczos three-term step.  Enqueued on `stream`; allocates nothing.  CSR handles launch
 * it with programmatic stream serialisation: consecutive steps on one stream overlap the tail of
 * one launch with the start of the next, which reads only the matrix arrays of the handle before
 * the preceding kernel has completed and every block after (so the matrix arrays must not be
 * written by work that is still in flight on `stream`). */
int polfed_fused_step(const polfed_ham* ham, int s, double p, double q, double r, double c,
                      const double* d_X, const double* d_Z, const double* d_V, double* d_Y,
                      void* stream);

/* 2 * n * s * sizeof(double): the two auxiliary blocks of PAPER.md:431. */
size_t polfed_filter_workspace_bytes(int64_t n, int s);
/* Workspace polfed_filter_apply needs for this handle: the value above for a CSR handle; for a
 * POLFED_FORMAT_TILED or _SECTOR handle and s in {16, 32}: 6 blocks (two b/partial pairs, V in
 * both row orders) plus (tiled) a per-CTA tile scratch and the tile counters. */
size_t polfed_filter_workspace_bytes_ham(const polfed_ham* ham, int s);

/* W = sum_{k=0..K} h_coeffs[k] T_k(H~) V,  H~ = (H - a)/b, by the Clenshaw recurrence
 * Eq. (51) PAPER.md:427-431:
 *     b_{K+1} = b_{K+2} = 0;  b_k = h_coeffs[k] V + 2 H~ b_{k+1} - b_{k+2}  (k = K..1);
 *     W = h_coeffs[0] V + H~ b_1 - b_2
 * as exactly K sparse products (max(K-1,0) + 1 launches of the fused kernel, plus one scaled
 * copy b_K = c_K V), on two rotating auxiliary blocks in d_work (pointer swap only, Fig. 5).
 * K >= 0.  h_coeffs: K+1 HOST doubles, read before return.  d_work holds
 * polfed_filter_workspace_bytes_ham(ham, s) bytes.  d_W must not overlap d_V or d_work.
 * b > 0 required (POLFED_ERANGE).  Enqueued on `stream`; allocates nothing; does not
 * synchronise.  On a POLFED_FORMAT_TILED or _SECTOR handle with s in {16, 32} the same recurrence
 * runs as K + 1 launches of the sweep kernel (see POLFED_FORMAT_TILED).  On a CSR handle with
 * n * s <= 262144 (configs 1 and 2: a fused launch is far shorter than the launch latency) the K
 * steps run inside one persistent kernel per 384 steps: a single CTA with both blocks in shared
 * memory for n * s <= 4096, else a cooperative grid with a grid barrier between the steps. */
int polfed_filter_apply(const polfed_ham* ham, double a, double b, int K, const double* h_coeffs,
                        int s, const double* d_V, double* d_W, void* d_work, void* stream);

/* Same operation on HOST blocks: takes device blocks from the library's own stream-ordered
 * memory pool (one per device, created on first use and never trimmed, so that later calls
 * reuse the blocks instead of allocating; the device's default pool is left alone), copies h_V
 * up, runs polfed_filter_apply, copies W down into h_W, returns the blocks to the pool,
 * synchronises.  The end-to-end entry. */
int polfed_filter_apply_host(const polfed_ham* ham, double a, double b, int K,
                             const double* h_coeffs, int s, const double* h_V, double* h_W,
                             void* stream);

/* ------------------------------------------------------------------------------------------
 * Filter parameters (host only).
 * ------------------------------------------------------------------------------------------ */

/* Delta-filter coefficients Eq. (32)-(33) PAPER.md:280-286 at sigma (unrescaled energy;
 * lambda~ = (sigma - a)/b must lie in (-1,1) else POLFED_ERANGE):
 *   c_0 = 1/chi, c_n = 2 T_n(lambda~)/chi, chi = 1 + 2 sum_{n=1..K} T_n(lambda~)^2   (R1).
 * Order: if rho_rescaled > 0 (states per unit rescaled energy at the target), K is
 * ceil(2.655 sqrt(1 - lambda~^2)/delta), delta = nev/(2 rho), Eq. (40), (42) PAPER.md:343-360,
 * refined by bisection on Eq. (41) in [K/2, 2K] with cutoff Omega = sin(2.655)/2.655 (R4);
 * otherwise K = K_in.  *K_out receives K; coeffs (capacity doubles, may be NULL to query K
 * only) receives K+1 values; capacity < K+1 gives POLFED_EINVAL with *K_out set. */
int polfed_filter_coeffs(double a, double b, double sigma, int nev, double rho_rescaled, int K_in,
                         int* K_out, double* h_coeffs, int capacity);

/* ------------------------------------------------------------------------------------------
 * Spectral bounds and the eigen-solver.
 * ------------------------------------------------------------------------------------------ */

/* Extremal Ritz values of n_steps scalar Lanczos steps with full reorthogonalisation started
 * from d_v0 (n doubles, any nonzero vector; normalised internally) -- PAPER.md:86-125 (Eq. 1-6),
 * 276-278, 462.  Outputs (any may be NULL): *emin, *emax the extremal Ritz values,
 * *a = (hi+lo)/2, *b = (1+margin)(hi-lo)/2 (Eq. 31 widened by `margin`, R5; margin < 0
 * means the default 0.01).  Ritz values lie inside the spectrum, so a and b are computed from
 * the extremal Ritz values moved outwards by their residual norms beta_{m+1} |z_m| (Eq. 6, 16;
 * zero once they have converged); *emin, *emax are the Ritz values themselves.  This is a
 * HEURISTIC, not an enclosure: the residual only guarantees SOME eigenvalue within that distance of
 * the Ritz value, not that E_max <= theta_max + residual.  With too few steps on a spectrum with
 * thin tails the true extremes can lie outside [a - b, a + b]; polfed_filter_apply then grows like
 * cosh(K acosh|x|) on those levels.  polfed_block_lanczos_eigs detects that (POLFED_ERANGE);
 * callers of polfed_filter_apply who need a guarantee should pass an enclosure of their own (e.g.
 * a Gershgorin bound) as a, b.
 * n_steps <= 0 means 60 (R6); it is clipped to n.  Allocates
 * (n_steps+1) x n doubles of device scratch and frees it; synchronises `stream`. */
int polfed_spectrum_bounds(const polfed_ham* ham, int n_steps, const double* d_v0, double margin,
                           void* stream, double* emin, double* emax, double* a, double* b);

/* Kernel polynomial method, PAPER.md:310-337 (Eq. 35-39): the density of states that sizes the
 * filter window (Eq. 40-42) when the Gaussian estimate Eq. (34) is not good enough (R7).
 *
 * polfed_kpm_moments: mu_m = (1/s) sum_{r<s} <r| T_m(H~) |r>, m = 0..n_moments-1 (Eq. 37-38), with
 * H~ = (H - a)/b and T_m by the Chebyshev recurrence Eq. (28)-(30) -- one fused sparse product and
 * one block dot product per moment.  d_R: n x s row-major fp64 DEVICE block of the random vectors
 * |r> (iid entries of zero mean and unit variance, drawn by the caller: no RNG crosses the ABI;
 * not modified); s in {1,2,4,8,16,32}; d_work: polfed_kpm_workspace_bytes(n, s, n_moments) bytes
 * of DEVICE scratch, 16-byte aligned; h_moments: n_moments doubles on the HOST.  mu_0 estimates the
 * dimension (the series integrates to it).  More than 32 vectors: call again and average.
 * Synchronises `stream`.  Errors: POLFED_EINVAL (NULL, s, n_moments < 1, alignment),
 * POLFED_ERANGE (b <= 0 or non-finite a, b). */
size_t polfed_kpm_workspace_bytes(int64_t n, int s, int n_moments);
int polfed_kpm_moments(const polfed_ham* ham, double a, double b, int n_moments, int s,
                       const double* d_R, void* d_work, double* h_moments, void* stream);
/* Host only: rho(E~) = [mu_0 g_0 + 2 sum_{m>=1} mu_m g_m T_m(E~)] / (pi sqrt(1 - E~^2)), Eq. (36),
 * with the Jackson kernel g_m of Eq. (39), at n_points rescaled energies in (-1, 1) (else
 * POLFED_ERANGE); rho is in states per unit rescaled energy, the unit polfed_filter_coeffs takes. */
int polfed_kpm_dos(const double* h_moments, int n_moments, const double* e_rescaled, int n_points,
                   double* rho);

/* The two tall-skinny products of the full reorthogonalisation (Eq. 9, 11 PAPER.md:147-153; cost
 * O(M^2 D)), exported so that they can be tested and timed on their own:
 *   polfed_block_gram:    C_j = Q_j^T B      for j < n_panels   (C: n_panels x s x s, row-major)
 *   polfed_block_update:  B = beta B + alpha sum_j Q_j C_j
 * Q_j = d_Q + j * panel_stride doubles, each n x s row-major like B; s in {1,2,4,8,16,32}; all
 * pointers DEVICE, 16-byte aligned, panel_stride >= n*s when there is more than one panel (else
 * POLFED_EINVAL, nothing is launched).  Every sum runs in a fixed order (bit-reproducible).
 * variant: 0 = the library's choice (fp64 tensor-core mma for s >= 8), 1 = the shared-memory FMA
 * kernel, 2 = tensor cores (s >= 8 only, else the FMA kernel).  Enqueued on `stream`; scratch for
 * the per-CTA partial sums comes from the library's stream-ordered pool (see
 * polfed_filter_apply_host). */
int polfed_block_gram(int s, int64_t n, const double* d_Q, int n_panels, int64_t panel_stride,
                      const double* d_B, double* d_C, int variant, void* stream);
int polfed_block_update(int s, int64_t n, const double* d_Q, int n_panels, int64_t panel_stride,
                        const double* d_C, double alpha, double beta, double* d_B, void* stream);

/* polfed_block_gram for callers that must not allocate device memory.
 *
 * Who needs it: a solver that has given all free HBM to its Krylov basis V_{1:m} (PAPER.md:469, 619:
 * the basis is the dominant memory), so that one more cudaMalloc -- or growth of the library's
 * scratch pool, which polfed_block_gram draws from -- fails; a process held to a fixed device-memory
 * budget by its scheduler or an MPS limit; a latency-bound loop that cannot take the device-wide
 * synchronisation the CUDA allocator may impose.  This entry point calls no cudaMalloc, cudaFree,
 * pool or other allocating routine.  Same arguments, same result layout and the same fixed-order
 * (bit-reproducible) sums as polfed_block_gram; the caller still owns d_Q, d_B and d_C.
 *
 * The per-CTA partial sums live in ONE array of POLFED_STATIC_GRAM_DOUBLES doubles (4 MiB) that is
 * part of the library's device image: every GPU that loads libpolfed.so holds those 4 MiB until the
 * process exits, whether or not this function is ever called.
 *   - Limit: n_panels * s * s <= POLFED_STATIC_GRAM_DOUBLES (s = 32: 512 panels; s = 16: 2048), else
 *     POLFED_ERANGE and nothing is launched.  Split a longer panel list over several calls.  When the
 *     grid polfed_block_gram would use needs more partial sums than fit, a smaller grid is taken:
 *     the result then differs from polfed_block_gram's in the last bits (another summation order),
 *     and is still the same on every run.
 *   - The first call on each device looks up the array's device address (cudaGetSymbolAddress, with
 *     that device current) and keeps it; make that first call outside any stream capture.
 *   - All calls share the array and it keeps whatever the last call left.  Nothing in it has to start
 *     at zero: each call overwrites every slot it later reads.  For the same reason two calls that
 *     run on the GPU at the same time (different streams, or different host threads on different
 *     streams) race on it and both results are garbage -- order them on one stream or with events.
 * Errors: POLFED_EINVAL (s, negative sizes, variant, NULL, a pointer not 16-byte aligned, overlapping
 * panels), POLFED_ERANGE (the limit above), POLFED_ECUDA (address lookup or launch failed). */
#define POLFED_STATIC_GRAM_DOUBLES 524288
int polfed_block_gram_static(int s, int64_t n, const double* d_Q, int n_panels, int64_t panel_stride,
                             const double* d_B, double* d_C, int variant, void* stream);

typedef struct {
  double tol;             /* absolute bound on ||H x - lambda x||; <= 0: 1e-8 * max(|E_min|,|E_max|) */
  int32_t max_krylov_dim; /* <= 0: 5 nev + 8 s rounded up to a multiple of s (R10), capped by n and by free memory */
  int32_t check_every;    /* block steps between convergence checks; <= 0: adaptive (R9) */
  int32_t K_override;     /* > 0: polynomial order; else Eq. (42)+(41) with the density of states
                             selected by `dos` (R7) */
  int32_t bounds_steps;   /* <= 0: 60 */
  double bounds_margin;   /* < 0: 0.01 */
  double a, b;            /* b > 0: rescaling parameters given, no Lanczos bounds run */
  int32_t sigma_is_rescaled; /* nonzero: sigma is the rescaled target lambda~ in (-1,1) (R8) */
  int32_t dos;            /* POLFED_DOS_GAUSSIAN (0): Eq. (34) from Tr H, Tr H^2;
                             POLFED_DOS_KPM (1): Eq. (35)-(39) */
  int32_t kpm_moments;    /* KPM: Chebyshev moments N; <= 0: 75 */
  int32_t kpm_vectors;    /* KPM: columns R of d_kpm_block, a positive multiple of 4 (paper: 100) */
  const double* d_kpm_block; /* KPM: n x kpm_vectors row-major DEVICE block of iid zero-mean
                             unit-variance entries drawn by the caller (no RNG crosses the ABI) */
  int32_t window_levels;  /* levels N the filter window of Eq. (40)-(41) is sized for.  <= 0: the
                             paper's rule, N = nev ("contains exactly N_ev eigenvalues"),
                             plus max(2, 10 %) (R4).  Larger N = lower order K; must be >= nev.
                             Measured on config 3 (nev = 100, s = 16): the Krylov dimension that
                             block Lanczos needs stays near 4.6 nev once the window holds <= 2 nev
                             levels, so N = 2 nev halves K and the time */
} polfed_options;
enum { POLFED_DOS_GAUSSIAN = 0, POLFED_DOS_KPM = 1 };

typedef struct {
  double a, b, lambda_rescaled, e_min, e_max, tol;
  int32_t K, block_steps, krylov_dim, n_converged, n_checks;
  int32_t K_gaussian;             /* order the Gaussian density of states gives (0 if not evaluated) */
  int64_t sparse_products;        /* fused launches, all phases */
  double seconds_bounds, seconds_filter, seconds_reorth, seconds_qr;
  double seconds_projected_eig;   /* dense eigen-decompositions of H_L and of the H-projection */
  double seconds_extraction, seconds_total;
  double rho_gaussian, rho_kpm;   /* states per unit rescaled energy at the target (0: not evaluated) */
  int32_t K_kpm;                  /* order the KPM density of states gives (0 if not evaluated) */
  int32_t nev_window;             /* levels the filter window is sized for: nev + max(2, 10 %), or
                                     options->window_levels */
  double seconds_dos;             /* moments of the density-of-states estimate */
  int64_t products_without_v;     /* of sparse_products: filter launches whose coefficient is exactly 0 and
                                     that therefore skip the read of V (R22; about half of them when the
                                     target is the middle of the interval) */
} polfed_report;

/* The nev eigenpairs of H nearest sigma (Sec. 4.6 steps 1-6):
 *   1. a, b from polfed_spectrum_bounds (first column of d_V0 as start) unless given;
 *   2. K from Eq. (40)-(42) with the Gaussian density of states Eq. (34), or with the KPM
 *      density Eq. (36) (options->dos = POLFED_DOS_KPM: the moments of polfed_kpm_moments over
 *      the caller's random block, the Jackson-damped series of polfed_kpm_dos at the target),
 *      unless K_override; the report carries both orders when both are evaluated;
 *   3. block Lanczos on P(H~) (Fig. 4): W = P(H~) V_k by polfed_filter_apply,
 *      A_k = V_k^T W, full reorthogonalisation against V_1..V_k (twice), W = V_{k+1} B_{k+1}
 *      by CholeskyQR2 (R17);
 *   4. at a check: eigen-decomposition of H_L (cuSOLVER syevd), the nev+s largest Ritz values,
 *      back-map u = V_{1:m} t (Eq. 43), Rayleigh-Ritz of H itself in span(u) (R21), residuals
 *      ||H x - E x||; stop when the nev extracted pairs nearest sigma all have residual <= tol
 *      (a converged pair farther away never stands in for an unconverged nearer one) and lie in
 *      the main lobe of the filter, P(lambda~_i) > Omega = 0.17613 (R4, R11).  The window is
 *      sized for nev + max(2, 10 %) levels so that a density estimate a few per cent off still
 *      leaves nev levels inside.
 * d_V0: n x s start block (need not be orthonormal; full column rank required).
 * Outputs: h_evals[nev] ascending, d_evecs n x nev row-major (column j pairs with h_evals[j]),
 * h_residuals[nev]; report may be NULL.  Returns POLFED_ENOCONV (outputs hold the best nev
 * pairs found) if max_krylov_dim is reached first, POLFED_EBREAKDOWN on a rank-deficient block,
 * POLFED_EWINDOW as soon as all nev + s (rounded up) extracted pairs are converged while fewer than
 * nev of them lie in the main lobe (the density of states was overestimated, so K is too high and
 * the window too narrow: the outputs are the nev converged eigenpairs nearest sigma, possibly not
 * contiguous; call again with a lower K_override or a larger window_levels), and POLFED_ERANGE when
 * a Rayleigh-Ritz value of H falls outside [a - b, a + b]: the bounds of step 1 are extremal Ritz
 * values moved outwards by their residuals and a margin -- a heuristic, NOT an enclosure (R5) -- and
 * a spectrum that sticks out makes the filter grow without bound there.
 * Allocates the Krylov basis (max_krylov_dim + s columns) and scratch on the device;
 * synchronises `stream`. */
int polfed_block_lanczos_eigs(const polfed_ham* ham, double sigma, int nev, int s, const double* d_V0,
                              const polfed_options* options /* may be NULL: all defaults */,
                              double* h_evals, double* d_evecs, double* h_residuals,
                              polfed_report* report, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* POLFED_H */

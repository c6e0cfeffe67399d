/* ftlm.h - C ABI of the B200-native FTLM hot path (arxiv/paper_2605_26261, PAPER.md).
 *
 * What the library computes: the matrix-free, row-wise gather y = H v (Eq. 12,
 * L97-L109) of the spin-1/2 Heisenberg Hamiltonian H = sum_b J_b s_i.s_j - h sum_i s^z_i
 * (Eq. 1; per-bond J_b and the Zeeman term are DESIGN.md readings 4-5) restricted to
 * one S^z sector, the state-to-index map it needs in two forms - the compressed lookup table
 * "CLT" (L148-L183, Alg. 2) and combinatorial ranking "CR" (L121-L146, Alg. 1) - fused with
 * the Lanczos recursion it drives (L45), plus the host-side tridiagonal eigensolve and FTLM
 * trace assembly (Eqs. 4-9).
 *
 * Conventions
 *  - Bit k of a label = 1 <=> site k up (Eq. 11); N_up = N/2 + M_z (Eq. 17).
 *  - Sector basis = labels with popcount N_up in ascending order; indices are 0-based
 *    int64_t, labels uint64_t; "not in the sector" = -1 (Alg. 2 step 2).
 *  - Every function returns FTLM_OK (0) or a positive error code; nothing throws across the
 *    ABI; ftlm_last_error() gives the thread-local message of the last failure.
 *  - "d_" arguments are DEVICE pointers, "h_" arguments (and all plain arrays of
 *    ftlm_create / ftlm_thermo / ftlm_tridiag_eig) are HOST pointers.  The library never
 *    takes ownership of a caller buffer.  Vectors hold ftlm_dim() elements of the handle's
 *    precision (float or double), densely packed.
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls
 *    documented "asynchronous" only enqueue work on it.
 *  - One GPU per handle.  There is no CPU fallback: without a CUDA device every device call
 *    fails with FTLM_ECUDA.
 */
#ifndef FTLM_H
#define FTLM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ftlm_ctx ftlm_ctx;

enum { FTLM_OK = 0, FTLM_EINVAL = 1, FTLM_ENOMEM = 2, FTLM_ECUDA = 3, FTLM_EUNSUPPORTED = 4 };
/* State-to-index strategies: the paper's compressed lookup table (Alg. 2), combinatorial ranking (Alg. 1,
 * L121-L146), and Lin's two half-system tables (L119: index = Ja[n >> h] + Jb[n & (2^h - 1)], h = N / 2, in the same
 * ascending-label order; N <= 48; served by the thread-per-row kernel only - the paper's own Lin kernel is its
 * comparison row kernel, "roughly half the throughput of the CLT-based variant"). */
enum { FTLM_INDEX_CLT = 0, FTLM_INDEX_CR = 1, FTLM_INDEX_LIN = 2 };
enum { FTLM_FP32 = 0, FTLM_FP64 = 1 };

/* Kernel variants selectable with ftlm_set_option("kernel", ...).
 * ROW  = one thread per row, every row unranked, per-bond loop (the paper's launch shape, L105,
 *        L136, L203), kept as the plain in-library baseline.
 * ROWG = the same per-bond loop with the row state the north_star describes: a thread owns 8 consecutive rows,
 *        unranks the first (L136) and steps to the next seven with a Gosper-style same-popcount successor; a lane's
 *        rows are 32 contiguous bytes, so the vector streams stay coalesced.  Single vector (no batch).
 * TML  = B200 design: label split into top/middle/low parts, one CTA per top part with the tile
 *        staged in shared memory and per-class neighbour tables. */
enum { FTLM_KERNEL_AUTO = 0, FTLM_KERNEL_ROW = 1, FTLM_KERNEL_ROWG = 2, FTLM_KERNEL_TML = 3 };

/* ---- handle ------------------------------------------------------------------------------ */

/* Build the sector tables on `device` (A0/A1 of SURVEY 8(a)): binomials C(n,k) (= D_c of
 * Eq. 16 at d = 2), bond masks and couplings, and in CLT mode the table of (M_b, C_b) pairs of
 * L150-L154 / Eq. 18.  All array arguments are host pointers and are copied.
 *   N in [1, 62]; 0 <= bond_i[b] != bond_j[b] < N (duplicates are legal and add); N_up in
 *   [0, N]; n_bonds in [0, 4096].  CLT needs N <= 32, LIN needs N <= 48.
 * Errors: FTLM_EINVAL (bad argument), FTLM_EUNSUPPORTED (CLT with N > 32, LIN with N > 48),
 *         FTLM_ENOMEM (table does not fit), FTLM_ECUDA (no device / CUDA failure). */
int ftlm_create(ftlm_ctx** out, int N, int n_bonds, const int32_t* bond_i, const int32_t* bond_j,
                const double* J, double h, int N_up, int index_mode, int precision, int device);

/* Free the handle and everything it owns (tables, chain workspace).  NULL is accepted. */
int ftlm_destroy(ftlm_ctx* ctx);

/* Sector dimension C(N, N_up). */
int64_t ftlm_dim(const ftlm_ctx* ctx);

/* Options: "kernel" (FTLM_KERNEL_*), "batch" (1, 2, 4: chains ftlm_lanczos / ftlm_lanczos_host advance together on
 * interleaved vectors, L207; default 1; rebuilds the tile split and the windows for rows of that many values),
 * "plan_batch" (0 = follow "batch"; else build the plans for that many chains even when fewer run),
 * "tml_low_bits" / "tml_mid_bits" / "tml_split" = w | m << 8 (split of the TML kernels, 0 = auto),
 * "graph" (1 = ftlm_chain_steps captures two consecutive fused steps - three with "lazy_norm" - into a CUDA graph
 * once and replays it; same kernels, same arithmetic, fewer launches: for the launch-bound small sectors; falls back
 * to direct launches if a graph call fails; read-only "graph_launches", "graph_failed"); "persistent" (1 =
 * ftlm_lanczos runs a sector whose three work vectors fit shared memory - read-only "persistent_fits" - with ONE
 * launch for all R chains: one CTA per chain, vectors resident in shared memory for the whole chain); multi-pass H.v of kernel TML (DESIGN.md
 * 6.4-6.5): "passb" (1 = bonds that leave the tile go to PASS-B window passes; default 0),
 * "passb_lo_min" / "passb_smax" / "passb_ctas" (window planner: lowest label position, largest
 * window, CTAs per SM tried first; 0 = auto), "tmlr" (1 = in-tile pass by the TMLR kernel when its
 * plan exists), "tmlr_unij" (0 = never use the uniform-J form), "lazy_norm" (1 = no separate
 * normalisation pass in a chain: the TMLR pass forms q_{j+1} while staging; needs "tmlr"), "allow_unverified" / "autotune_mask" (ftlm_autotune: run candidates without a device record / only
 * the candidates whose bit is set).  The checked and emulation builds (not the release library) also accept the test
 * hooks "debug_pass_mask", "debug_item_first", "debug_item_count" (run only some passes / tiles / items of a non-fused
 * H.v).  FTLM_EINVAL on unknown key/value, FTLM_EUNSUPPORTED
 * when the requested kernel / split cannot be built for this sector.  ftlm_get_option also answers
 * read-only keys: "sm_count", "autotuned", "tml_w", "tml_m", "tml_smem", "tml_ctas_per_sm",
 * "tml_threads", "tml_tiles", "tml_n_ll|mm|ml|tt|tm|tl", "tml_bclass:<b>", "tmlr_available",
 * "tmlr_smem", "tmlr_n_ll|mm|ml|g", "tmlr_unij_used", "lazy_norm_ok", "passb_windows", "passb_bonds",
 * "passb_lo<k>", "passb_mask<k>", "passb_nbonds<k>", "passb_items<k>", "passb_ctas_used". */
int ftlm_set_option(ftlm_ctx* ctx, const char* key, int64_t value);
int64_t ftlm_get_option(const ftlm_ctx* ctx, const char* key);

/* Bytes of index-table memory on the device (CLT: 8*ceil(2^N/32), Eq. 21; CR: the small tables). */
int64_t ftlm_table_bytes(const ftlm_ctx* ctx);

/* Copy CLT blocks [b0, b0+nb) to host arrays (test hook for A1).  FTLM_EINVAL in CR mode. */
int ftlm_clt_read(ftlm_ctx* ctx, int64_t b0, int64_t nb, uint32_t* h_mask, uint32_t* h_count);

/* ---- index maps (L0) --------------------------------------------------------------------- */

/* d_idx[k] = sector index of d_labels[k] with the handle's index mode, -1 if the label is not
 * in the sector (CLT: Alg. 2; CR: Alg. 1).  Asynchronous. */
int ftlm_index_of(ftlm_ctx* ctx, const uint64_t* d_labels, int64_t n, int64_t* d_idx, void* stream);

/* d_labels[k] = label of sector index d_idx[k] (the inverse map, L136); indices outside
 * [0, dim) give UINT64_MAX.  Asynchronous. */
int ftlm_state_of(ftlm_ctx* ctx, const int64_t* d_idx, int64_t n, uint64_t* d_labels, void* stream);

/* d_idx[(r*n_bonds + b)] for rows row0 <= row0+r < row0+nrows: index of the source state that
 * bond b couples row row0+r to (the "lookup[n_ij]" of Eq. 12), or -1 if the bond's spins are
 * parallel.  Computed by the SAME device code path as the H.v kernel selected by "kernel".
 * Asynchronous. */
int ftlm_neighbors(ftlm_ctx* ctx, int64_t row0, int64_t nrows, int64_t* d_idx, void* stream);

/* ---- Hamiltonian action (L1) ------------------------------------------------------------- */

/* y = H v (Eq. 12).  d_v, d_y: dim elements of the handle's precision, d_y != d_v and
 * non-overlapping.  Asynchronous on `stream`. */
int ftlm_apply_H(ftlm_ctx* ctx, const void* d_v, void* d_y, void* stream);

/* Host-buffer variant: copies h_v to the device, applies H, copies y back; synchronous. */
int ftlm_apply_H_host(ftlm_ctx* ctx, const void* h_v, void* h_y);

/* ---- start vectors ----------------------------------------------------------------------- */

/* d_v = normalised Gaussian start vector r of this sector under `seed`: the counter-based
 * generator specified in DESIGN.md section 4 (element t depends only on seed, N_up, r, t);
 * generated and normalised in FP64, rounded once to the handle's precision.  Asynchronous. */
int ftlm_fill_random(ftlm_ctx* ctx, uint64_t seed, int r, void* d_v, void* stream);

/* ---- fused Lanczos chain (L2) ------------------------------------------------------------ */

/* Begin a chain: q_1 = d_q1 (copied; need not be normalised) or, if d_q1 == NULL, the seeded
 * vector ftlm_fill_random(seed, r).  Allocates the handle's three work vectors on first use.
 * Asynchronous. */
int ftlm_chain_begin(ftlm_ctx* ctx, const void* d_q1, uint64_t seed, int r, void* stream);

/* Enqueue `nsteps` more fused Lanczos steps (L45): per step one fused
 * H.v pass  y = H q_j - beta_{j-1} q_{j-1}  with FP64-accumulated <q,y>, <y,y>, <q,q>, and one
 * pass q_{j+1} = (y - alpha_j q_j)/beta_j.  alpha, beta stay on the device; after a breakdown
 * (beta_j <= tol*max(|alpha_k|, beta_k), tol = 1e-5 FP32 / 1e-12 FP64) or once min(n, dim)
 * steps are done the remaining launches are no-ops.  At most FTLM_MAX_STEPS per chain.
 * Asynchronous. */
int ftlm_chain_steps(ftlm_ctx* ctx, int nsteps, void* stream);

/* Synchronise `stream` and copy out the coefficients: alpha[0..m_eff), beta[0..m_eff-1).
 * `cap` = capacity of h_alpha (and of h_beta).  h_m_eff receives the number of steps done. */
int ftlm_chain_end(ftlm_ctx* ctx, double* h_alpha, double* h_beta, int cap, int* h_m_eff, void* stream);

/* Batched chains (the paper's batched Lanczos, L207, L309, Table 3 footnote L325): begin `batch` (1, 2 or 4) chains
 * r0 .. r0 + batch - 1 from their seeded start vectors on interleaved work vectors q[t][batch]; every fused pass
 * then computes the row state and every neighbour index once for all of them.  ftlm_chain_steps advances the whole
 * batch; each chain has its own alpha, beta and breakdown state, and its coefficients are bit-identical to those of
 * the same chain run alone with the same kernel, tile split and windows (option "plan_batch" builds a single chain's
 * plans for a batch's geometry).  batch > 1 runs the ROW kernel, or the TML in-tile pass with or without PASS-B
 * windows (the register-table TMLR pass and lazy normalisation are single-vector); batch must not exceed the batch
 * the handle's plans were built for (options "batch" / "plan_batch"; FTLM_EINVAL).  Asynchronous. */
int ftlm_chain_begin_batch(ftlm_ctx* ctx, uint64_t seed, int r0, int batch, void* stream);

/* ftlm_chain_end for the batch in progress: chain b -> h_alpha[b*cap ...], h_beta[b*cap ...], h_m_eff[b]. */
int ftlm_chain_end_batch(ftlm_ctx* ctx, double* h_alpha, double* h_beta, int cap, int* h_m_eff, void* stream);

/* Run `nsteps` steps with CUDA events around every kernel and return the average device time
 * (ms) of the fused H.v kernel and of the normalisation kernel.  Synchronous; for bench.py. */
int ftlm_chain_profile(ftlm_ctx* ctx, int nsteps, void* stream, double* ms_hv, double* ms_norm);

/* Choose the H.v kernel configuration of the handle by measurement on the device (DESIGN.md
 * section 7.1).  Each candidate computes y = H v for one seeded random vector and is compared on
 * the device with the thread-per-row kernel (Eq. 12 with Alg. 1 / Alg. 2 as printed, L105-L173);
 * candidates beyond the H.v tolerance (1e-5 FP32, 1e-12 FP64, norm-relative), or whose first three
 * fused Lanczos steps deviate from the thread-per-row kernel's alpha, beta by more than 1e-4 / 1e-9,
 * are rejected; the others are timed over `reps` fused steps (CUDA events) and the fastest is left
 * selected.  report (host, caller-owned, may be NULL): JSON list of {name, valid, relerr,
 * fused_dev, ms, windows}.  Allocates and frees 3 vectors of dim elements and uses the handle's
 * chain workspace (any chain in progress is lost).  Synchronous.  FTLM_EUNSUPPORTED if no
 * candidate is valid (the handle keeps its previous selection). */
int ftlm_autotune(ftlm_ctx* ctx, int reps, char* report, int report_cap, void* stream);

#define FTLM_MAX_STEPS 1024

/* Whole sector: R chains from seeded starts r = 0..R-1, n_steps each, then the Ritz pairs.
 * Host outputs (caller-owned): alpha[R][n_steps], beta[R][n_steps], m_eff[R],
 * theta[R][n_steps], weight[R][n_steps] (weight = s_{k,1}^2, L45); entries beyond m_eff[r] are
 * zero.  theta/weight may be NULL.  Synchronous. */
int ftlm_lanczos(ftlm_ctx* ctx, uint64_t seed, int R, int n_steps, double* h_alpha, double* h_beta,
                 int* h_m_eff, double* h_theta, double* h_weight, void* stream);

/* Same with caller-provided HOST start vectors h_q1[R][dim] (handle precision): each is copied
 * host->device inside the call (end-to-end path of bench.py). */
int ftlm_lanczos_host(ftlm_ctx* ctx, const void* h_q1, int R, int n_steps, double* h_alpha,
                      double* h_beta, int* h_m_eff, double* h_theta, double* h_weight, void* stream);

/* ---- host-only parts (A8, A9) ------------------------------------------------------------ */

/* Eigenvalues theta[m] (ascending) of the symmetric tridiagonal T(alpha[m], beta[m-1]) and
 * weights weight[k] = (first component of the normalised eigenvector k)^2 (L45).  FP64. */
int ftlm_tridiag_eig(int m, const double* alpha, const double* beta, double* theta, double* weight);

/* FTLM trace assembly, Eqs. 7-9 (L61-L74).  Sector s has dim[s], magnetisation Mz[s],
 * multiplicity mult[s] (2 for M_z > 0, reading 15), R[s] chains; chain c of sector s has
 * m_eff[off+c] Ritz pairs stored at theta/weight[(off+c)*stride ...], off = sum of R over
 * earlier sectors.  Outputs per temperature T[i]: E_ref (scalar, = min theta),
 * Zs = Z*exp(E_ref/T), E = <H>, C = (<H^2>-<H>^2)/T^2, chi = g^2 sum Mz^2 Z_M/(T sum Z_M). */
int ftlm_thermo(int n_sec, const int64_t* dim, const double* Mz, const double* mult, const int* R,
                int stride, const int* m_eff, const double* theta, const double* weight, int nT,
                const double* T, double g, double* E_ref, double* Zs, double* E, double* C,
                double* chi);

/* ---- host diagnostics ------------------------------------------------------ */

/* Ghost diagnostic of one chain (section 3.2): theta/weight as ftlm_tridiag_eig; ell[k] = min_j |theta_k -
 * theta^(1)_j| with T^(1) = T without its first row and column (Cullum-Willoughby, Eq. 25); ghost[k] = 1
 * iff ell[k] < tau, tau = C_tau * 2^-24 * (theta_max - theta_min) (FP32 unit roundoff for both precisions, L262);
 * cluster[k] = id (ascending from 0) of the cluster of Ritz values chained by gaps <= tau and cluster_weight[k] the
 * summed weight of that cluster (L270); F[k] = sum_{k' <= k} weight[k'] (Eq. 23).  All arrays host, length m,
 * caller-owned; ell, ghost, cluster, cluster_weight, F, tau may be NULL.  m = 1: ell = +inf. */
int ftlm_ghost_diagnostic(int m, const double* alpha, const double* beta, double C_tau, double* theta,
                          double* weight, double* ell, int* ghost, int* cluster, double* cluster_weight,
                          double* F, double* tau);

/* Eq. 22 (L225-L228): samples[s*nT + i] = estimate of an observable from seed set s at temperature i;
 * mean[i] and sigma[i] = sqrt((1/N_s) sum_s (O_s - mean)^2). */
int ftlm_sigma_emp(int n_seeds, int nT, const double* samples, double* mean, double* sigma);

/* L230: sigma_theo[i] = |O[i]| / sqrt(Z_eff[i]), Z_eff = Tr exp(-(H - E_0)/T) (= Zs of ftlm_thermo). */
int ftlm_sigma_theo(int nT, const double* O, const double* Z_eff, double* sigma);

const char* ftlm_last_error(void);
const char* ftlm_version(void);

#ifdef __cplusplus
}
#endif
#endif /* FTLM_H */

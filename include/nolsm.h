/* nolsm.h -- C ABI of the B200-native NOLSM hot path (arXiv 2205.12182).
 *
 * The library evaluates, one atom-block at a time, the density matrix
 *     D = 1/2 (I - sign(S^-1 H0 - mu I)) S^-1                          (Eq. 5)
 * with the non-orthogonal local submatrix method (per-submatrix form Eq. 8)
 * and the electronic energy E_elec = Tr(D H0) (Eq. 4).
 *
 * Inputs are the sparse H0, S and the scalar mu; outputs are D with the input
 * sparsity pattern and the scalar E_elec. Everything runs on one GPU (sm_100a).
 *
 * Conventions
 *   - Every pointer argument documented "host or device" may point to host memory (pageable or
 *     pinned) or to device memory of `cuda_device`; the library detects which. Device arrays are
 *     BORROWED until nolsm_destroy or the next nolsm_assemble and never freed by the library. Host
 *     arrays are copied during the call and may be released when it returns (for asynchronous
 *     outputs: after nolsm_energy returned). A D_vals in pinned host memory is filled by a copy enqueued behind the
 *     kernel; a D_vals in pageable host memory is filled by the first call that waits for the results (nolsm_energy, a
 *     getter, the next density_matrix call), so that the time limit is watched while the kernel runs.
 *   - Block-CSR: row i lists the atoms j with a block (i, j), ascending. Slot s = (i, j) holds the
 *     nb(i) x nb(j) block row-major; slot s starts at element blk_off[s] = sum over earlier slots of
 *     nb(i') * nb(j'). H0 and S share one pattern (the union of their patterns), which
 *     must be structurally symmetric with every diagonal block present.
 *   - Output layout: D_vals uses the same pattern and offsets; slot (i, j) holds (D_ji)^T, where block
 *     D_ji (rows of atom j, columns of atom i) is taken from submatrix i. The array is
 *     therefore D^T in block-CSR and row i is written by submatrix i alone (with options.combine: by the submatrix of the
 *     group atom i belongs to). D is not symmetrised.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = default stream).
 *   - All functions return a nolsm_status; none throws (every entry point catches what its host code may throw and
 *     returns NOLSM_ENOMEM / NOLSM_ECUDA with the text in nolsm_last_error), aborts or traps: a persistent kernel that overruns
 *     options.timeout_s, or in which a wait stalls (device watchdog), is stopped through an abort word and the call
 *     that waits for it returns NOLSM_ECUDA. Numerical failures of single
 *     submatrices are reported asynchronously: they set per-atom status bits (nolsm_get_atom_stats) and
 *     make nolsm_energy return NOLSM_ENOTSPD / NOLSM_ENOCONV after writing the result.
 */
#ifndef NOLSM_H
#define NOLSM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nolsm_ctx nolsm_ctx; /* opaque, owned by the library */

typedef enum {
    NOLSM_OK = 0,
    NOLSM_EINVAL = 1,   /* bad argument / malformed pattern */
    NOLSM_ECUDA = 2,    /* a CUDA call failed (nolsm_last_error has the text) */
    NOLSM_ENOMEM = 3,
    NOLSM_ESTATE = 4,   /* call out of order */
    NOLSM_ENOTSPD = 5,  /* some S_sub inverse iteration diverged or did not converge */
    NOLSM_ENOCONV = 6   /* some sign iteration hit max_sign_iters (result written, flagged) */
} nolsm_status;

enum { NOLSM_PREC_FP16_FP32 = 0, /* FP16 operands, FP32 accumulate, tcgen05 tensor cores */
       NOLSM_PREC_FP32 = 1 };    /* all-FP32 validation mode (FFMA, no tensor cores, no TF32) */
enum { NOLSM_DTYPE_F64 = 0, NOLSM_DTYPE_F32 = 1 };
enum { NOLSM_GEMM_AUTO = 0, NOLSM_GEMM_UMMA = 1, NOLSM_GEMM_SIMT = 2 };
enum { NOLSM_ENGINE_AUTO = 0, NOLSM_ENGINE_PERSISTENT = 1, NOLSM_ENGINE_ROUNDS = 2 };
enum { NOLSM_ITER_EQ6 = 0,       /* Eq. 6 as printed: S^-1 by the Schulz iteration, sign iteration on A = S^-1 H0 - mu I */
       NOLSM_ITER_LOWDIN = 1 };  /* symmetric form: Z = S^-1/2 by the coupled Newton-Schulz iteration, the same sign
                                    iteration on the symmetric Z H0 Z - mu I, D = Z 1/2 (I - X) Z; every iterate is symmetric
                                    (C-21). Persistent engine only. */
enum { NOLSM_MAT_NOTSPD = 1, NOLSM_MAT_NOCONV = 2 }; /* per-atom status bits */

/* Zero in any field selects the default given in brackets. */
typedef struct {
    int precision;           /* NOLSM_PREC_* [FP16_FP32] */
    int gemm_backend;        /* NOLSM_GEMM_* [AUTO: UMMA (tcgen05, persistent engine) for FP16_FP32, SIMT (FFMA, round engine) for FP32] */
    int max_inv_iters;       /* cap on Schulz inverse iterations [24] */
    int max_sign_iters;      /* cap on Newton-Schulz sign iterations, Eq. 6 [64] */
    float tol_inv;           /* stop when ||I - S Y||_F / sqrt(n) < tol_inv [2e-3 mixed, 1e-5 FP32] */
    float tol_sign;          /* stop when ||X^2 - I||_F / sqrt(n) < tol_sign [2e-3 mixed, 1e-5 FP32] */
    int power_iters_s;       /* power iterations for rho(S_sub) [persistent engine 3 (x 1.3 safety), round engine 6 (x 1.05)] */
    int power_iters_a;       /* power iterations for rho(A_sub) [persistent engine 6 (x 1.25 safety; more while the estimate is not
                                settled, nolsm_get_engine_counters out[38]), round engine 12 (x 1.05)] */
    double eps_filter;       /* block (j,i) enters N(i) iff max(|H0_ji|max, |S_ji|max) > eps_filter [0 = structural] */
    int batch_atoms;         /* workspace slots = submatrices resident at once [auto: persistent engine heavy_slots + max(12, heavy_slots),
                                at most 96; round engine ~16 waves of GEMM tiles] */
    size_t workspace_bytes;  /* cap on the library-owned dense workspace [auto] */
    int profile_every;       /* round engine, > 0: every k-th round runs eagerly with CUDA events around each launch [0 = off] */
    int engine;              /* NOLSM_ENGINE_* [AUTO: PERSISTENT (one kernel launch per density_matrix call, tcgen05 GEMMs) for the
                                FP16_FP32 path when every n_i <= 4096 and nb(i) <= 16; else ROUNDS (plain FFMA GEMMs, one CUDA
                                graph per iteration round): the validation engine] */
    int sign_scaled_iters;   /* persistent engine: the first k sign iterations run Eq. 6 on alpha X_k instead of X_k,
                                X_{k+1} = 1/2 (alpha X_k)(3I - (alpha X_k)^2), alpha = sign_scale > 1, which lifts small
                                eigenvalues 1.5 alpha x per step instead of 1.5 x and keeps the rest inside
                                [alpha (3 - alpha^2) / 2, 1]; two steps with the optimal scalings for that interval follow,
                                then plain Eq. 6 until the convergence test passes (C-6b) [6; -1 = plain Eq. 6] */
    float sign_scale;        /* alpha of the scaled steps, 1 < alpha < sqrt(3) [1.5] */
    int combine;             /* persistent engine: one submatrix for several columns. 0 = one submatrix per atom;
                                1 = greedy groups under the cubic criterion Eq. 9 (L87); 2 = under Eq. 10 (L91): predicted runtime
                                n^3 / r(n) with the measured multiplication rate r(n) of nolsm_set_perf_table, linearly interpolated
                                (without a table: the tile-step model ceil(n16/256)^2 ceil(n16/64), C-19) [0] */
    int combine_max_dim;     /* a group's union index set may not exceed this dimension [2048] */
    int combine_max_members; /* atoms per group at most [16] */
    int combine_max_candidates; /* candidates examined per seed atom, by descending overlap with the seed's index set [24] */
    int iteration;           /* NOLSM_ITER_* [EQ6] */
    int symmetric_tiles;     /* persistent engine: products of symmetric commuting matrices (the Schulz iterates; every product of
                                the Loewdin form) multiply only the tiles on and above the diagonal of the tile grid and mirror
                                them [0 = on; -1 = off: every tile is multiplied] */
    int heavy_slots;         /* persistent engine: submatrices inside the GEMM chains at once [0 = auto: L2 size / (3.5 n^2 FP16)] */
    int mu_trials;           /* nolsm_find_mu, persistent engine: trial mu evaluated per pass on the resident S_sub^-1, A0 [1 = bisection:
                                a trial after the first costs ~3/4 of a pass and K trials gain log2(K + 1) bits, so K = 1 needs the
                                least work per bit (measured: bench.py other_configs.cfg1.mu_search); max 8] */
    double timeout_s;        /* persistent engine: time limit of one kernel, counted from its launch. The call that waits for the
                                results (nolsm_energy, any getter) stops a kernel that runs longer; inside the kernel a hot wait
                                (pipeline stages, accumulators) that lasts timeout_s / 10 (at least 2 s) or an idle wait (tile
                                records) that lasts timeout_s (at least 20 s) counts as a stall and stops the kernel too. The abort
                                of any kernel launched since the last wait is reported by that wait, also when later calls on
                                the context (a series of nolsm_density_matrix_range) went through [300] */
    int transposed_tiles;    /* persistent engine: the tiles of a ragged last row block (r < 256 rows left) are computed transposed,
                                C^T = B^T A^T, so the MMA's M = 256 runs over full columns and its N = r over the rows that exist,
                                instead of M = 256 (or 128) over r rows [0 = on; -1 = off] */
    int tuning[8];           /* engine tuning words with measured defaults (profiles/r02_persist.md); they carry no meaning for a
                                user of the method, are not part of the stable interface, and should stay zero. Persistent
                                engine: [0] claim lead: a CTA pair claims its next tile when its TMA producer is this many
                                k-blocks from the end of the current one [14]; [1] slot scan order of the tile schedulers,
                                1 = every pair from slot 0, 2 = every pair from its own slot [auto: 2 for mean dimensions up
                                to 768]; [2] / [3] L2 eviction priority of the TMA operand loads / of the TMA stores of the GEMM
                                results, 1 evict_first, 2 evict_last, 3 normal [1 / 2]; [4..7] unused */
} nolsm_options;

typedef struct {
    int64_t n_atoms;
    int64_t n_batches;            /* engine rounds of the last density_matrix call */
    int64_t dim_min, dim_max;
    double dim_mean;
    int64_t sum_inv_iters, sum_sign_iters;
    int64_t gemms_executed;       /* square GEMMs actually run, summed over submatrices */
    double flops_useful;          /* FLOP of the executed tiles on true dimensions: sum_i 2 n_i^3 * (full GEMMs_i + the executed share of
                                     the symmetric ones) */
    double flops_padded;          /* same with tile-padded dimensions (what the tensor cores executed) */
    int64_t n_notspd, n_noconv;
    double gather_bytes, scatter_bytes; /* algorithmic bytes of the last density_matrix call */
    int64_t n_units;              /* dense submatrices evaluated per call (== n_atoms without combination); dim_min / dim_max /
                                     dim_mean describe these */
    int64_t gemms_symmetric;      /* of gemms_executed: symmetric products that multiplied the upper triangle of tiles only; they
                                     count (ntm + 1) / (2 ntm) of 2 n^3 in flops_useful (the share of tiles executed) */
    double flops_paper;           /* sum_i 2 n_i^3 * gemms_i with every product counted in full (PAPER.md:L156 knows no symmetric ones) */
} nolsm_stats;

/* Layout check for bindings that restate the structs above (paper_2205_12182_b200/binding.py does): the version is bumped
 * whenever a field of nolsm_options / nolsm_stats or the meaning of an existing argument changes, and the two sizes are the
 * library's own sizeof. A binding compares all three with its own at load time and refuses a stale libnolsm.so instead
 * of silently misreading every option behind the first changed field. Needs no context and no GPU. */
#define NOLSM_ABI_VERSION 6
int nolsm_abi_version(void);
size_t nolsm_sizeof_options(void);
size_t nolsm_sizeof_stats(void);

/* Creates a context on `cuda_device`. opt may be NULL. */
int nolsm_create(nolsm_ctx** out, int cuda_device, const nolsm_options* opt);

/* a0: takes the block-CSR pattern and values of H0 and S, validates it, builds the
 * index sets N(i), dimensions n_i, and the batch plan; uploads what lives on the host.
 *   atom_nb  int32[n_atoms]     basis functions per atom (> 0)                 host or device
 *   row_ptr  int64[n_atoms+1]                                                  host or device
 *   col_idx  int32[nnzb]        ascending inside each row                      host or device
 *   H0_vals, S_vals             val_dtype[blk_off[nnzb]]                        host or device
 * Returns NOLSM_EINVAL for unsorted columns, a non-symmetric pattern, a missing diagonal block,
 * atom_nb <= 0 or null pointers. Synchronises `cuda_stream` before returning. */
int nolsm_assemble(nolsm_ctx* ctx, int64_t n_atoms, const int32_t* atom_nb, const int64_t* row_ptr,
                   const int32_t* col_idx, const void* H0_vals, const void* S_vals, int val_dtype,
                   void* cuda_stream);

/* a1-a7 for all atoms: gather, Schulz inverse, spectral scaling, Newton-Schulz sign (Eq. 6),
 * convergence tests, D columns, scatter and energy partials. The work is ordered after everything
 * already enqueued on `cuda_stream`, and `cuda_stream` is made to wait for it. Persistent engine: the
 * call enqueues ONE kernel and returns. Round engine: the call returns once the last round has been
 * enqueued (the host replays one CUDA graph per round and reads a device-written progress counter).
 *   D_vals   d_dtype[blk_off[nnzb]]   host or device; blocks outside every N(i) are zeroed. */
int nolsm_density_matrix(nolsm_ctx* ctx, double mu, void* D_vals, int d_dtype, void* cuda_stream);

/* Same for atoms [atom_begin, atom_end) only; other rows of D_vals are left untouched. If
 * e_partial_host is not NULL the call synchronises and stores sum of e_i over the range. With combine every group
 * that has a member in the range is evaluated and serves its members inside the range (a group that straddles a range
 * boundary is evaluated once per range it touches). */
int nolsm_density_matrix_range(nolsm_ctx* ctx, double mu, int64_t atom_begin, int64_t atom_end, void* D_vals,
                               int d_dtype, double* e_partial_host, void* cuda_stream);

/* Eq. 4: synchronises the stream of the last density_matrix call, finishes pending device-to-host
 * copies and returns E_elec = sum_i e_i over the atoms evaluated by that call. */
int nolsm_energy(nolsm_ctx* ctx, double* e_elec);

int nolsm_destroy(nolsm_ctx* ctx);

/* ---- diagnostics used by the parity tests and the benchmark ---- */

/* Tr(D S) of the last density_matrix call (the chemical potential is iterated until the electron count
 * is right): sum over the evaluated atoms i of q_i = sum_{j in N(i)} <D_ji, S_ji>, accumulated in FP64 in the scatter
 * step. q_atom_out (host, nullable) receives the q_i of the evaluated range. Synchronises. */
int nolsm_electron_count(nolsm_ctx* ctx, double* n_elec, double* q_atom_out);

/* Tr(D(mu_j) S) for n_mu (1..8) trial chemical potentials in ONE pass over the atoms (mu is iterated
 * until the electron count is right; S_sub^-1 and A0 = S_sub^-1 H_sub do not depend on mu): every submatrix is gathered
 * and inverted once, then the sign chain (Eq. 6) and the traces run once per trial mu on the resident A0 - mu_j I
 * (C-20). No D is written. n_elec_out[j] = Tr(D(mu_j) S), e_out[j] (nullable) = Tr(D(mu_j) H0); host arrays.
 * Persistent engine only. Synchronises. NOLSM_ENOTSPD / NOLSM_ENOCONV as for nolsm_energy. */
int nolsm_electron_counts(nolsm_ctx* ctx, const double* mu, int n_mu, double* n_elec_out, double* e_out, void* cuda_stream);

/* Chemical-potential search for |Tr(D(mu) S) - n_target| <= tol_n on [mu_lo, mu_hi]; stops also when
 * the bracket is narrower than tol_mu or max_evals (0 = 40) trial mu were evaluated. Tr(D S) never decreases with mu;
 * NOLSM_EINVAL if n_target is not bracketed. Persistent engine: the end points, then options.mu_trials equidistant trial mu
 * per pass (nolsm_electron_counts: the bracket shrinks by mu_trials + 1 per pass, the gather and the inverse are done once
 * per pass), and one final nolsm_density_matrix call at the mu reported. Round engine: bisection, one full call per trial.
 * On return D_vals (host or device, as for nolsm_density_matrix) holds D(mu_out), n_out = Tr(D(mu_out) S), evals_out the
 * trial mu evaluated; nolsm_energy and nolsm_get_stats refer to the final call. */
int nolsm_find_mu(nolsm_ctx* ctx, double n_target, double mu_lo, double mu_hi, double tol_n, double tol_mu, int max_evals,
                  void* D_vals, int d_dtype, void* cuda_stream, double* mu_out, double* n_out, int* evals_out);

/* The group (unit) atom `atom` belongs to after nolsm_assemble (C-19; without combine the group is the atom
 * itself): its members in joining order (seed first), the union index set (ascending atom ids) that the group's one
 * dense submatrix is built on, and that submatrix's dimension. Call with NULL arrays to query the two counts. */
int nolsm_get_group(nolsm_ctx* ctx, int64_t atom, int32_t* members_out, int32_t* n_members_inout, int32_t* set_out,
                    int32_t* n_set_inout, int32_t* dim_out);

/* p(n) of Eq. 10 ("the matrix multiplication performance p(n) of the GPUs is measured for different
 * matrix sizes n and interpolated"): count measured points, dimensions n[] strictly ascending in 1..8192, rates in TFLOP/s
 * (rounded to integer GFLOP/s). combine = 2 then compares predicted runtimes n^3 / r(n), r linearly interpolated between
 * neighbouring points and constant outside the table, in integer arithmetic (csrc/grouping.cpp). Takes effect at the next
 * nolsm_assemble; count = 0 removes the table. workloads/pn_b200.json holds the table measured on B200 with
 * `python bench.py --pn-sweep`. Host arrays. */
int nolsm_set_perf_table(nolsm_ctx* ctx, const int32_t* n, const double* tflops, int count);

/* N(i) (ascending atom ids) and n_i. atoms_out may be NULL to query the count; capacity in *n_inout. */
int nolsm_get_index_set(nolsm_ctx* ctx, int64_t atom, int32_t* atoms_out, int32_t* n_inout, int32_t* dim_out);

/* Runs the gather kernel for one atom and copies the dense submatrix the atom is evaluated on (row-major, tight) to
 * host memory: n_i x n_i on N(i), or with combine the group's submatrix on its union index set (dimension and set from
 * nolsm_get_group; FP16 only). which: 0 = T(S), 1 = T(H0). out_fp16 != 0 -> uint16 FP16 bits, else float. */
int nolsm_gather_submatrix(nolsm_ctx* ctx, int64_t atom, int which, int out_fp16, void* out_host);

/* The same gather as nolsm_gather_submatrix (FP16 output), for callers that must not allocate device memory.
 *
 * Who that is: a host program that has already handed all of the GPU's memory to its own pool (a tensor framework's
 * caching allocator, an MD code's arena) so that any further cudaMalloc fails; and a program that inspects submatrices
 * while other work is in flight on the GPU, because cudaMalloc / cudaFree synchronise the whole device and would stall
 * until, for example, a running density-matrix kernel of several seconds has finished. nolsm_gather_submatrix does one
 * cudaMalloc + cudaFree per call and gathers into the context's workspace; this entry point calls no cudaMalloc,
 * cudaFree or any other allocating routine, and leaves the workspace and the results of the last density_matrix call
 * untouched.
 *
 * What it uses instead: the gather kernel writes the padded dense T(S) and T(H0) (rows of n16 = n rounded up to 16
 * FP16 values, 16-byte stores) into a scratch array that is part of the library image: a fixed `static __device__`
 * array of 2 * NOLSM_NOALLOC_MAX_DIM^2 FP16 values = 16 MiB. Every GPU on which the library is loaded holds these
 * 16 MiB from the moment the library's device code is loaded there until the process exits, whether or not this
 * function is ever called. The requested matrix is then copied, tight, from the scratch array to `out`.
 *   atom       the atom; with options.combine the submatrix of the atom's group is gathered (dimension: nolsm_get_group)
 *   which      0 = T(S), 1 = T(H0)
 *   out        uint16 FP16 bits, n x n row-major, tight; memory the CALLER owns. Device memory: the kernel and the copy
 *              are enqueued on `cuda_stream` and the call returns without waiting. Host memory: the call waits for the
 *              stream before it returns.
 * Limit: a submatrix whose padded dimension n16 exceeds NOLSM_NOALLOC_MAX_DIM is refused with NOLSM_EINVAL (the text of
 * nolsm_last_error names both numbers); nothing is launched. Persistent engine only (NOLSM_ESTATE otherwise).
 *
 * First call on a device: it looks up the device address of the scratch array (cudaGetSymbolAddress) and raises the
 * kernel's shared-memory limit, once per device and process. Make that first call outside any stream capture; later
 * calls only launch one kernel and one 2-D copy.
 *
 * Sharing: there is ONE scratch array per GPU, shared by every context and every thread of the process. Calls whose GPU
 * work can overlap (different streams, or different contexts on one device) overwrite each other's scratch and return
 * garbage: keep them on one stream, or order them with events. The array keeps whatever the previous call left in it;
 * that is harmless, because each call writes every element it later copies out (the kernel zero-fills its row strips
 * before placing the blocks), so nothing has to be cleared between calls. */
#define NOLSM_NOALLOC_MAX_DIM 2048
int nolsm_gather_submatrix_noalloc(nolsm_ctx* ctx, int64_t atom, int which, void* out, void* cuda_stream);

int nolsm_get_stats(nolsm_ctx* ctx, nolsm_stats* out);

/* Per-atom results of the last density_matrix call for atoms [atom_begin, atom_begin + count); any
 * output pointer may be NULL. Host arrays. */
int nolsm_get_atom_stats(nolsm_ctx* ctx, int64_t atom_begin, int64_t count, int32_t* dims, int32_t* inv_iters,
                         int32_t* sign_iters, int32_t* status, int32_t* gemms, float* residual, double* e_atom);

/* Per-launch device times of the rounds sampled by options.profile_every during the last
 * density_matrix call (those rounds run eagerly on one stream with CUDA events recorded around each
 * launch; all other rounds replay the CUDA graph). FLOP and byte counts cover the sampled rounds only.
 *   out[0..2]   gather:  total ms, launches, algorithmic bytes (source blocks read + dense FP16/FP32 written)
 *   out[3..6]   GEMM:    total ms, launches, useful FLOP (2 n^3 per executed GEMM), tile-padded FLOP
 *   out[7..9]   D columns + scatter: total ms, launches, algorithmic bytes (X and Y columns read, D row written, H0 row read)
 *   out[10..11] other kernels (mat-vecs, state, flags): total ms, launches
 *   out[12]     submatrices gathered in the sampled rounds;  out[13] kernel launches of the whole call
 * After a call served by the persistent engine (one kernel, nolsm_get_engine_counters out[0] = 1) the same slots
 * describe that kernel and cover the whole call: out[3] = its duration in ms (CUDA events on its stream), out[4] = 1,
 * out[5..6] FLOP of all its GEMMs; out[0..2], out[7..9] and out[10..11] are the side tasks inside it (gather; D columns
 * + scatter; refill + first Schulz step): busy ms summed over the side groups, tasks, algorithmic bytes;
 * out[12] = submatrices of the call, out[13] = 1.
 * n must be >= NOLSM_PROFILE_LEN. Synchronises the stream. */
#define NOLSM_PROFILE_LEN 14
int nolsm_get_profile(nolsm_ctx* ctx, double* out, int n);

/* Counters of the persistent engine for the last density_matrix call (all zero after a round-engine call).
 *   out[0] 1 = persistent engine ran;  out[1] kernel duration in ms (CUDA events on its stream);
 *   out[2] kernel duration from the device clock (first scheduler start to last scheduler end), ms;
 *   out[3] GEMM tiles executed (256 x bn, one per CTA pair);  out[4], out[5] tile-scheduler idle / busy
 *   time summed over the CTA pairs, ms;  out[6] claim overshoots;  out[7] slots;  out[8] CTA pairs;
 *   out[9 + k], out[17 + k], out[25 + k]  side tasks of kind k (1 refill, 2 gather, 3 elementwise steps,
 *   4 D columns + scatter, 5 W columns of the Loewdin form): busy ms summed over side groups, algorithmic bytes, tasks;
 *   out[33..35] where the MMA-issuing warps (one per CTA pair) spent the kernel, ms summed over the pairs: waiting for a
 *   tile record, waiting for a free accumulator (= for the epilogue), inside k-loops (operand waits + issue);
 *   out[36..37] the tile schedulers, ms summed over the pairs: waiting for a free entry of the record ring (= for the
 *   completion of the tile four back), waiting for the producer's claim point;
 *   out[38] power-iteration steps for rho(A) beyond options.power_iters_a, summed over the submatrices: the iteration
 *   goes on (up to 24 steps) while the estimate still grows by more than 5 % per step or its growth rises from one step to
 *   the next, the mark of an eigenvalue outside the bulk that the fixed step count would underestimate.
 *   n must be >= NOLSM_COUNTERS_LEN. Synchronises. */
#define NOLSM_COUNTERS_LEN 39
int nolsm_get_engine_counters(nolsm_ctx* ctx, double* out, int n);

/* HBM-bound side tasks timed alone: which = 0 the gather of every submatrix of the assembled system (a1),
 * which = 1 the D columns + scatter + energy of every atom (a6-a7, on whatever the slots hold). The device functions of
 * the persistent kernel, one 128-thread side group per CTA, `reps` launches between CUDA events. ms_out = mean time of one
 * launch, bytes_out = algorithmic bytes of one launch (source blocks read + dense FP16 rows written; D written + H0, S,
 * P and Y columns read). Invalidates the results of the last density_matrix call. Persistent engine only. */
int nolsm_side_task_bandwidth(nolsm_ctx* ctx, int which, int reps, double* ms_out, double* bytes_out);

const char* nolsm_last_error(const nolsm_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* NOLSM_H */

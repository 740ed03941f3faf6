/*
 * ctqmc.h — C ABI of the B200-native CT-HYB local-trace library (libctqmc_b200.so).
 *
 * The library evaluates, for many Monte-Carlo configurations per call, the local impurity trace of the
 * hybridisation-expansion solver of arXiv:2010.08482 (ComCTQMC),
 *
 *     w_loc(C) = sum_{q0} Tr P_{beta-tau_L}(q_L) F_{alpha_L}(q_{L-1}) ... F_{alpha_1}(q_0) P_{tau_1}(q_0)      (Eq. 65)
 *
 * with P_tau(q) = diag(exp(-tau E_q[n])) the propagator in the eigenbasis of H_loc, F_alpha(q) the dense
 * sector-to-sector blocks of c_f / c^dag_f, and s_alpha(q) the sector map with its "zero sector"
 * (PAPER.md:534); and the lazy-trace upper bound built from submultiplicative norms of the factors.
 *
 * Everything on the path runs in sm_100a CUDA kernels; there is no CPU fallback.  All functions return 0 on success or
 * a negative CTQMC_ERR_* code; on error nothing has been written to the outputs.  `ctqmc_last_error()` gives the text.
 *
 * Concurrency: a handle owns one scratch arena, so batch calls on the SAME handle must be issued one after the other (they may
 * be on different streams as long as the second is enqueued after the first has completed); different handles are independent.
 *
 * Pointer conventions are stated per argument: HOST = ordinary host memory, DEVICE = device memory of the GPU the
 * impurity was loaded on (e.g. a torch tensor's data_ptr()).
 */
#ifndef CTQMC_H
#define CTQMC_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CTQMC_OK               0
#define CTQMC_ERR_ARG         -1   /* null pointer, bad size, inconsistent description */
#define CTQMC_ERR_OOM         -2   /* device or host allocation failed */
#define CTQMC_ERR_CUDA        -3   /* a CUDA call or kernel launch failed */
#define CTQMC_ERR_UNSUPPORTED -4   /* valid request the library does not implement (e.g. a device that is not sm_100) */

/* Per-configuration status values written to `status[b]`. */
#define CTQMC_STATUS_OK        0
#define CTQMC_STATUS_VANISHING 1   /* no start sector survives the sector map: w_loc = 0 structurally */
#define CTQMC_STATUS_INVALID   2   /* symbol out of range, tau decreasing or outside [0, beta): outputs are NaN */

/* Schedules for ctqmc_set_option(CTQMC_OPT_SCHEDULE, ...). */
#define CTQMC_SCHEDULE_THIN    0   /* default: start each string at its smallest sector (exact by cyclicity of the trace) */
#define CTQMC_SCHEDULE_LITERAL 1   /* start at q0 and carry dim(q0) columns, the literal order of Eq. 65 */

#define CTQMC_OPT_SCHEDULE     1
#define CTQMC_OPT_PANEL_WIDTH  2   /* columns carried per work unit: 8, 16, 32 (0 = automatic) */
#define CTQMC_OPT_TIMING       3   /* 1: record CUDA events around the phases of every batch call (see ctqmc_last_timing) */
#define CTQMC_OPT_PATH         4   /* which chain kernel family runs (CTQMC_PATH_*); results agree up to rounding */
#define CTQMC_OPT_SCRATCH_LIMIT 5  /* upper limit in bytes for the AUTOMATIC growth of the scratch arena (0 = 80 % of the free device
                                      memory).  A batch whose scratch exceeds the arena is evaluated in rounds of configurations;
                                      if not even one configuration fits, AUTO falls back from the grouped to the panel kernel and
                                      an explicit CTQMC_PATH_GROUPED request returns CTQMC_ERR_OOM */
#define CTQMC_OPT_SPLIT_SLICES 7   /* int8 slices per operand of CTQMC_PATH_SPLIT: 5 .. 8 (default 7); set before selecting the path */
#define CTQMC_OPT_ARENA_BYTES  6   /* allocate the scratch arena NOW with exactly this many bytes and never grow it (0 = back to
                                      automatic growth).  PAPER.md:574: "we pre-allocate ... and develop our own memory allocator
                                      which can work asynchronously with that block": after this call no batch call allocates,
                                      frees or synchronises; a batch that does not fit is cut into rounds, and CTQMC_ERR_OOM is
                                      returned BEFORE anything is enqueued if one configuration alone does not fit */

/* Kernel families for CTQMC_OPT_PATH.  AUTO: the small-sector kernel (whole path in one launch, operator store in shared
 * memory) when every sector has at most 16 states; else, when a panel of the largest sector fits in shared memory, the
 * step-synchronous grouped GEMM kernel for batches of 64 configurations or more and the persistent shared-memory panel
 * kernel for smaller ones; else the large-sector tiled GEMM kernel (one launch per chain position).  Every path only enqueues:
 * scratch and launch shapes are sized on the host from upper bounds it knows (n_configs, n_ops, max_len, the sector dimensions),
 * the actual counts stay on the device.
 * ctqmc_bound_batch: segment_len 1 uses tables only (one fused launch for small real impurities); other segment lengths run
 * the panel kernel family, or the large-sector one when the sectors do not fit in shared memory. */
#define CTQMC_PATH_AUTO        0
#define CTQMC_PATH_PANEL       1
#define CTQMC_PATH_LARGE       2
#define CTQMC_PATH_SMALL       3
#define CTQMC_PATH_GROUPED     4   /* step-synchronous grouped GEMM: strings that apply the same block share one GEMM per chain position */
#define CTQMC_PATH_SPLIT       5   /* large-sector path with every chain step evaluated by split-precision (Ozaki-type) int8 tensor-core
                                      products, exact up to 7 * slices - 1 bits below the largest entry of each operand row / column
                                      ("mixed-precision matrix-multiplication kernel"); complex impurities; never chosen by AUTO */

/* Diagnostic environment variables, read when an impurity is loaded or a path is selected (results do not depend on them
 * beyond rounding): CTQMC_LARGE_TMA=0 stages the large-sector kernel's tiles with cp.async instead of TMA; CTQMC_SMALL_V1=1
 * runs real small impurities on the element-per-lane small kernel that complex ones use; CTQMC_SMALL_G=8|16|32 sets that
 * kernel's lanes per configuration. */

typedef struct ctqmc_impurity ctqmc_impurity;   /* opaque; created by ctqmc_load_impurity, destroyed by ctqmc_free_impurity */

/*
 * Description of the impurity in the eigenbasis of H_loc (sector decomposition and per-sector
 * diagonalisation are done once at initialisation, by the caller).  All pointers are HOST memory; the library copies
 * what it needs and the caller keeps ownership.
 */
typedef struct {
  int32_t        n_sectors;    /* Q >= 1 (Eq. 64) */
  const int32_t* dim;          /* [Q] sector dimensions, each >= 1 */
  const double*  energy;       /* [sum dim] eigenvalues of H_loc, sector-major; any finite values */
  int32_t        n_symbols;    /* A: number of operator symbols alpha; for c / c^dag: alpha = 2*flavour + (1 if creation) */
  int32_t        is_complex;   /* 0: block data are doubles; 1: interleaved (re, im) pairs of doubles */
  int64_t        n_blocks;     /* number of non-zero sector-to-sector blocks; at most one per (symbol, src) */
  const int32_t* blk_symbol;   /* [n_blocks] alpha */
  const int32_t* blk_src;      /* [n_blocks] q          */
  const int32_t* blk_dst;      /* [n_blocks] s_alpha(q);  (symbol, src) pairs without a block map to the zero sector */
  const int64_t* blk_offset;   /* [n_blocks] element offset of the block inside blk_data */
  const void*    blk_data;     /* per block: column-major dim[dst] x dim[src]; element (m,n) = < m in dst | O_alpha | n in src > */
} ctqmc_impurity_desc;

/*
 * A batch of configurations in CSR form.  A configuration is a time-ordered operator string
 * (alpha_1, tau_1), ..., (alpha_L, tau_L) with 0 <= tau_1 <= ... <= tau_L < beta; index 0 acts first (rightmost in
 * PAPER.md:519, Eq. 63).  The library applies no time-ordering sign (the caller passes ordered operators).
 * L = 0 is legal and yields Z = sum_n exp(-beta E_n).
 */
typedef struct {
  int64_t        n_configs;    /* B >= 0 */
  const int64_t* offset;       /* [B+1], offset[0] = 0, non-decreasing */
  const int32_t* symbol;       /* [n_ops] */
  const double*  tau;          /* [n_ops] */
  int64_t        n_ops;        /* HOST value: length of symbol / tau (= offset[B]).  The device forms cannot read offset[B] without
                                  waiting for the device, so the caller states it; a configuration whose offsets leave [0, n_ops]
                                  gets status 2 instead of an out-of-bounds read.  Host forms: 0 = take offset[B] */
  int32_t        max_len;      /* HOST value: no configuration has more than this many operators (sizes the per-chain-position
                                  launch loops and the scratch); longer configurations get status 2.  0 = unknown: the library
                                  falls back to n_ops, which is correct but enqueues one step per operator of the WHOLE batch --
                                  state it.  Host forms compute it from the offsets */
} ctqmc_batch;

/* Load an impurity onto CUDA device `device`: copies dims / energies, builds the routing table s_alpha(q), the padded
 * row-major operator store and the per-block norm tables (row-norm^2, Frobenius, spectral) with device kernels.
 * Errors: CTQMC_ERR_ARG for Q < 1, dim < 1, non-finite energy, block indices out of range, duplicate (symbol, src). */
int ctqmc_load_impurity(const ctqmc_impurity_desc* desc, int device, ctqmc_impurity** out);

void ctqmc_free_impurity(ctqmc_impurity* imp);

/* Tuning knobs (CTQMC_OPT_*); affects subsequent batch calls on this handle.  Results are independent of them up to
 * floating-point rounding. */
int ctqmc_set_option(ctqmc_impurity* imp, int option, int64_t value);

/*
 * Evaluate w_loc (Eq. 65) for every configuration of the batch.  `batch` fields and all outputs are DEVICE pointers.
 * The call only enqueues work on `cuda_stream` (a cudaStream_t, NULL = default stream) and returns; outputs are valid
 * once the stream reaches that point; it never waits for the device and never reads anything back.  The scratch arena is one
 * device block: with CTQMC_OPT_ARENA_BYTES it is fixed and no call ever allocates; otherwise it grows -- before anything is
 * enqueued, and only when a call needs more than every earlier one (allocation synchronises the device).
 *
 *   mant    [B][2]  (re, im) mantissa; im = 0 for real impurities; max(|re|,|im|) in [1,2), or (0,0) for an exact zero,
 *                   or (NaN, NaN) for status 2
 *   exp2    [B]     w_loc = (mant_re + i mant_im) * 2^exp2   (running exponent: long chains neither overflow nor underflow)
 *   survive [B][Q]  or NULL: 1 iff the sector string starting at q0 never hits the zero sector
 *   status  [B]     CTQMC_STATUS_*
 */
int ctqmc_trace_batch(ctqmc_impurity* imp, double beta, const ctqmc_batch* batch,
                      double* mant, int64_t* exp2, uint8_t* survive, int32_t* status, void* cuda_stream);

/*
 * Upper bounds on |w_loc| from submultiplicative norms.  With the cyclic factorisation
 * A_i = P_{Delta_i}(q_i) F_{alpha_i}(q_{i-1}), Delta_i = tau_{i+1} - tau_i, Delta_L = beta - tau_L + tau_1, and segments
 * G_j of `segment_len` consecutive factors (0 = the whole chain, i.e. one segment):
 *
 *   norm_kind 0 (Frobenius):  B(q0) = sqrt(d_min) * prod_j ||G_j||_F
 *   norm_kind 1 (spectral):   B(q0) = d_min * prod_j u_j, u_j a rigorous upper estimate of ||G_j||_2:
 *                             segment_len 1:  u_i = exp(-Delta_i Emin(q_i)) sigma_max(F_{alpha_i}(q_{i-1}));
 *                             otherwise:      u_j = min(||G_j||_F, prod_{i in segment j} u_i)  (||XY||_2 <= ||X||_2 ||Y||_2 and
 *                             ||G||_2 <= ||G||_F; an iterative estimate of ||G_j||_2 approaches it from below and is not used).
 *                             sigma_max comes from a power iteration at load time, which approaches it from below: where the
 *                             iteration has not converged to 1e-10 (it converges exactly for c / c^dag blocks, whose F^H F is a
 *                             projector) the rigorous upper estimate min(||F||_F, sqrt(||F||_1 ||F||_inf)) is used instead, so the
 *                             result is always an upper bound
 *
 * with d_min the smallest sector dimension along the string; the configuration's bound is sum_{q0} B(q0).  All values
 * are rounded outward by (1 + 2^-40), so bound >= |w_loc| holds for the returned numbers.
 *
 *   bound_mant [B], bound_exp2 [B]                   bound = mant * 2^exp2, mant in [1,2) or 0
 *   sector_bound_mant [B][Q], sector_bound_exp2 [B][Q]   or NULL: B(q0), zero where q0 does not survive
 *   status [B]                                        as for ctqmc_trace_batch
 *
 * Conditioning signal: the ratio bound / |w_loc| of the Frobenius bound (norm_kind 0, segment_len 1) to the trace of the same
 * batch is an upper estimate of the cancellation in the final sector sum and chain products (reading A8: the oracle's
 * kappa); a caller that sees ratios beyond ~1e6 has lost that many digits of the 1e-9 bar and should label its sectors with every
 * conserved quantum number.
 */
int ctqmc_bound_batch(ctqmc_impurity* imp, double beta, const ctqmc_batch* batch, int norm_kind, int segment_len,
                      double* bound_mant, int64_t* bound_exp2, double* sector_bound_mant, int64_t* sector_bound_exp2,
                      int32_t* status, void* cuda_stream);

/*
 * Host-buffer convenience forms: identical results, but `batch` fields and all outputs are HOST pointers.  The library
 * copies the batch to the device, runs the same kernels, copies the results back and synchronises the stream before
 * returning (this is the end-to-end path bench.py times).  If every buffer passed to ctqmc_trace_batch_host is page-locked
 * (cudaHostAlloc / cudaHostRegister / torch pin_memory) the copies go straight from / to the caller's memory, and on the
 * small-sector path batches of 32768 configurations or more are cut into four chunks whose host-to-device copies (on an
 * internal stream) overlap the previous chunk's kernel; pageable buffers go through the library's pinned staging area.
 */
int ctqmc_trace_batch_host(ctqmc_impurity* imp, double beta, const ctqmc_batch* batch,
                           double* mant, int64_t* exp2, uint8_t* survive, int32_t* status, void* cuda_stream);
int ctqmc_bound_batch_host(ctqmc_impurity* imp, double beta, const ctqmc_batch* batch, int norm_kind, int segment_len,
                           double* bound_mant, int64_t* bound_exp2, double* sector_bound_mant, int64_t* sector_bound_exp2,
                           int32_t* status, void* cuda_stream);

/* Counters of the most recent batch call on this handle, summed over its rounds and (host form) chunks (HOST outputs;
 * synchronises the stream it ran on):
 * stats[0] = surviving strings, stats[1] = work units, stats[2] = kernels launched by the call,
 * stats[3] = real multiply-adds executed by the chain kernel (padded tiles included),
 * stats[4] = algorithmic real flops of the schedule executed (2 per real MAC, 8 per complex MAC, unpadded dims),
 * stats[5] = panel width (panel path) or lanes per configuration (small path), stats[6] = warps per team (panel path),
 * stats[7] = kernel family that ran (CTQMC_PATH_*), stats[8] = propagator exponentials evaluated (small path: sum over chain
 * steps of the sector dimension), stats[9] = bytes of the scratch arena. */
int ctqmc_last_stats(ctqmc_impurity* imp, int64_t stats[10]);

/* With CTQMC_OPT_TIMING = 1: device time in milliseconds of the phases of the most recent batch call on this handle,
 * from CUDA events recorded on the call's stream (HOST output; synchronises that stream):
 * ms[0] = validate + route + binning kernels, ms[1] = chain kernel(s) ("matrix multiplication ... kernels",
 * with the propagator, rescale and trace fused), ms[2] = final reduction kernels, ms[3] = whole call.
 * CTQMC_ERR_ARG if timing was not enabled when the call was made. */
int ctqmc_last_timing(ctqmc_impurity* imp, double ms[4]);

/* FP64 peak of `device` in TFLOP/s, measured with register-resident loops of independent mma.sync m8n8k4 f64 (DMMA) and
 * of plain DFMA (no memory traffic; best of 3 after a warm-up).  The roofline denominator of bench.py: the driver's
 * MEASURED_PEAKS.json holds HBM and bf16 peaks only.  HOST outputs; synchronises. */
int ctqmc_measure_fp64_peak(int device, double* tflops_dmma, double* tflops_dfma);

/* ------------------------------------------------------------------------------------------------------------------------
 * Chain sets: the incremental, lazy local trace for many Markov chains at once.
 *
 * "we can store these subproducts in a data structure, e.g., a balanced binary tree or a skip-list ... requiring
 * O[log(k)] matrix multiplications rather than O(k)".  PAPER.md:542-548 (lazy trace): the random number of the Metropolis
 * test is drawn first; bounds from submultiplicative norms of the stored sub-products decide the move as early as possible,
 * start sectors being evaluated one at a time.  PAPER.md:560-574: many chains share one device, device memory is one
 * pre-allocated block, only asynchronous calls.  The paper defers the data structure to its Ref. [9]; readings F1-F4 of
 * DESIGN.md fix it:
 *
 *   F1  every chain owns a complete binary tree over a FIXED dyadic partition of [0, beta) into 2^depth leaves; node (l, i)
 *       stores, for every sector q that survives it, the evolution operator across its interval (propagators to both ends
 *       included) as a dense matrix with an integer and a real exponent, its target sector and its Frobenius norm;
 *   F2  a proposal dirties the leaves containing its times and their ancestors: at most max_edits * (depth + 1) nodes;
 *   F3  bound of a proposal without multiplying the dirty ancestors: B(q0) = sqrt(r) * prod ||U_node||_F over the cover of the
 *       time axis by the recomputed dirty leaves and the maximal clean subtrees, r = smallest sector dimension at its seams,
 *       rounded outward by (1 + 2^-40);
 *   F4  decision against the caller's threshold T on |w_new| (log2 T per chain): sum_q0 B(q0) <= T rejects at once; else the
 *       start sectors are evaluated exactly in order of decreasing bound, and with S the sum so far and R the sum of the
 *       remaining bounds, |S| - R > T accepts and |S| + R <= T rejects.  An accepted proposal is completed (all sectors), so
 *       its trace is returned.
 *
 * All chains advance in lock-step through the same launches; which chains still need work is decided on the device.  Every
 * call only enqueues on `cuda_stream`; nothing is read back and nothing is allocated after ctqmc_chains_create.
 * Sector dimensions up to 512 (dense nodes per chain: "the simulation drops the Markov chain if the memory
 * request is denied" -- here ctqmc_chains_create returns CTQMC_ERR_OOM with the size needed). */
typedef struct ctqmc_chains ctqmc_chains;

typedef struct {
  int64_t n_chains;        /* C >= 1 */
  int32_t depth;           /* the time axis is cut into 2^depth leaves (choose 2^depth ~ expansion order) */
  int32_t leaf_capacity;   /* operators one leaf can hold (1 .. 64); a proposal that overflows a leaf gets status 4 */
  int32_t max_edits;       /* inserted + removed operators per chain per proposal (1 .. 16); 4 covers a pair move */
  int32_t lazy_rounds;     /* start sectors evaluated one at a time (one round of launches each) before the remaining
                              sectors of still-undecided chains are evaluated together; 0 = all at once */
} ctqmc_chains_desc;

/* Proposed edits in CSR form, DEVICE pointers: chain c proposes edits [offset[c], offset[c+1]): operator (symbol, tau) is
 * inserted (kind = +1) or removed (kind = -1; it must be present with exactly this tau).  n_edits is a HOST value. */
typedef struct {
  const int64_t* offset;   /* [C+1] */
  const double*  tau;      /* [n_edits] */
  const int32_t* symbol;   /* [n_edits] */
  const int32_t* kind;     /* [n_edits] */
  int64_t        n_edits;
} ctqmc_edit_batch;

/* Per-chain status of a proposal */
#define CTQMC_CHAIN_OK          0
#define CTQMC_CHAIN_BAD_EDIT    2   /* tau outside [0, beta), symbol out of range, kind not +-1, too many edits, corrupt offsets */
#define CTQMC_CHAIN_NOT_FOUND   3   /* removal of an operator the chain does not hold */
#define CTQMC_CHAIN_LEAF_FULL   4   /* a leaf would hold more than leaf_capacity operators */

/* Allocates the chain set in ONE device block and builds the trees of the empty configuration (w_loc = Z). */
int ctqmc_chains_create(ctqmc_impurity* imp, double beta, const ctqmc_chains_desc* desc, void* cuda_stream, ctqmc_chains** out);
void ctqmc_chains_destroy(ctqmc_chains* chains);

/* Lazy evaluation of one proposal per chain (readings F3, F4); the chains are not modified.  DEVICE pointers:
 *   log2_threshold [C]  log2 of T (-inf accepts every non-vanishing proposal); NULL = -inf for every chain
 *   accept [C]          1 / 0;   decided_by [C]  0 = by the bound alone, 1 = after part of the sectors, 2 = after all
 *   n_sectors_evaluated [C]  start sectors whose exact term entered the decision (all of them when accepted)
 *   bound_mant / bound_exp2 [C]  sum_q0 B(q0) of the proposed configuration (NaN for a non-zero status)
 *   trace_mant [C][2] / trace_exp2 [C]  w_loc of the proposed configuration when accepted, else 0
 *   status [C]          CTQMC_CHAIN_*; a chain with non-zero status is not accepted */
int ctqmc_chains_propose(ctqmc_chains* chains, const ctqmc_edit_batch* edits, const double* log2_threshold, int32_t* accept,
                         int32_t* decided_by, int32_t* n_sectors_evaluated, double* bound_mant, int64_t* bound_exp2,
                         double* trace_mant, int64_t* trace_exp2, int32_t* status, void* cuda_stream);

/* Applies the most recent proposal of every chain c with mask[c] != 0 (DEVICE [C]; NULL = its accept flags): the proposed
 * operators become the configuration, the shadow nodes the stored sub-products (entries the lazy evaluation never needed
 * are multiplied now).  Committing swaps slot indices; nothing is copied. */
int ctqmc_chains_commit(ctqmc_chains* chains, const int32_t* mask, void* cuda_stream);

/* w_loc of every chain's current configuration from its stored root: mant [C][2], exp2 [C] (DEVICE). */
int ctqmc_chains_trace(ctqmc_chains* chains, double* mant, int64_t* exp2, void* cuda_stream);

/* HOST outputs; synchronises the stream of the most recent call: stats[0] = matrix products performed since creation,
 * stats[1] = bytes of the chain set's device block, stats[2] = kernels enqueued by the most recent call,
 * stats[3] = node slots per chain (stored + shadow + scratch). */
int ctqmc_chains_stats(ctqmc_chains* chains, int64_t stats[4]);

/* ------------------------------------------------------------------------------------------------------------------------
 * Reduced density matrix of the impurity.  PAPER.md:254, Eq. 27:
 *     rho_uv = (1 / beta) < int_0^beta w_loc(C, P_vu(tau)) / w_loc(C) dtau >,   P_vu = |v><u|,  u, v eigenstates of one sector,
 * "this integration is done analytically".  The call ADDS, for every configuration b with status[b] == 0 and
 * w_loc != 0, weight[b] times the configuration's estimator to `rho` ("matrix addition" kernel): per surviving
 * closed string one forward sweep that keeps every prefix product and one backward sweep that forms (G_i Y_i)_uv for every
 * interval between two operators.  Each configuration's contribution has unit trace.
 *
 *   batch                    as for ctqmc_trace_batch (DEVICE; max_len must be stated: it sizes the per-string scratch)
 *   w_mant [B][2], w_exp2 [B], status [B]   DEVICE: the outputs of ctqmc_trace_batch for the SAME batch
 *   weight [B] or NULL       DEVICE: e.g. the sign of the configuration (NULL = 1)
 *   rho                      DEVICE, ctqmc_density_size(imp) elements (doubles, or (re, im) pairs for complex impurities):
 *                            sector q at offset sum_{q' < q} dim[q']^2, column-major, element rho_uv at u + v * dim[q].
 *                            The caller zeroes it before the first call and divides by the number of samples afterwards.
 * Only enqueues on `cuda_stream`.  Sector dimensions up to 512; scratch (max_len * d_max^2 elements per string in flight) comes
 * from the handle's arena under the rules of ctqmc_trace_batch. */
int64_t ctqmc_density_size(const ctqmc_impurity* imp);
int ctqmc_density_batch(ctqmc_impurity* imp, double beta, const ctqmc_batch* batch, const double* w_mant, const int64_t* w_exp2,
                        const int32_t* status, const double* weight, double* rho, void* cuda_stream);

/* ctqmc_density_batch for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid it): same arguments, same arithmetic, same kernel, but the per-string scratch lives in a file-scope device array
 * of ctqmc_density_static_limit() = 64 MiB bytes (every GPU that loads the library holds it until the process exits) instead of
 * the handle's arena.  The call allocates and frees nothing on the device and only enqueues on `cuda_stream`.
 *   - A string needs (max_len + 5) * d_max^2 elements (x2 complex) + 2 * (max_len + 2) words of scratch; if that exceeds the
 *     limit the call returns CTQMC_ERR_UNSUPPORTED and enqueues nothing (config 2 at max_len 300: 0.2 MB per string; config 4
 *     does not fit -- use ctqmc_density_batch).  Fewer strings in flight than ctqmc_density_batch when the array is the limit.
 *   - The first call on a device resolves the array's device address (cudaGetSymbolAddress, once per device): make that call
 *     outside a graph capture.
 *   - Every call on a device shares the ONE array, which keeps the last call's contents (nothing in it has to start at zero:
 *     a string only reads what it has written; the kernel's work counter, a second static word, is zeroed by every call on
 *     its stream).  Calls that overlap on the GPU -- different streams, or this call concurrent
 *     with itself from two host threads -- RACE on it; order them on one stream or with events. */
int64_t ctqmc_density_static_limit(void);
int ctqmc_density_batch_static(ctqmc_impurity* imp, double beta, const ctqmc_batch* batch, const double* w_mant, const int64_t* w_exp2,
                               const int32_t* status, const double* weight, double* rho, void* cuda_stream);

/* Thread-local description of the last error on this thread ("" if none). */
const char* ctqmc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* CTQMC_H */

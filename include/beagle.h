/* beagle.h — C-ABI of the B200-native Beagle scoring library (libbeagle_b200.so).
 *
 * What it is: batched fitness evaluation ("scoring", Table 1) of a whole colony of
 * symbolic-regression programs. PAPER.md:63 (§2.4): "the individual is sent to the GPU once and
 * the aggregated fitness value is returned for the full batch of fitness cases"; at
 * most 1024 fitness cases, so that one model is aggregated on chip and never through global
 * memory; PAPER.md:40 (§2.2): populations are managed in batches when device memory is short;
 * PAPER.md:184 (§3.2): a program is a flat list of commands run on an operand stack (RPN);
 * the stack holds 32 entries; PAPER.md:200-294 (Table 3): command meanings and
 * operand order; "length (i.e., the number of GCL commands)".
 * Where the paper is silent the readings of DESIGN.md §3 (R1..R25) apply.
 *
 * Conventions
 *   - Every entry point is extern "C", takes plain pointers and sizes, never throws, never aborts.
 *   - "DEVICE" = pointer into CUDA device memory of the current device; "HOST" = host memory.
 *   - All pointers are borrowed for the duration of the enqueued work; the library never frees or
 *     keeps user memory. Scratch lives in a library-owned workspace (see beagle_reserve).
 *   - Calls enqueue work on `stream` (a cudaStream_t passed as void*, NULL = legacy default
 *     stream) and return without synchronising. Blocking: the host is blocked in exactly two
 *     cases, both "the library-owned workspace has to grow": (a) P is larger than every earlier P
 *     and than beagle_reserve's P_max (cudaDeviceSynchronize + cudaMalloc of the per-individual
 *     arrays); (b) the micro-op workspace is not known to hold the call, i.e. it is smaller than
 *     the worst case (516 records per individual) and no beagle_reserve(P_max, T_max) with
 *     P <= P_max covers it: the token total is then read back (one cudaStreamSynchronize of
 *     `stream`) and the workspace grown. After beagle_reserve(P_max, T_max), calls with P <= P_max
 *     and at most T_max tokens only enqueue and can be captured in a CUDA graph. Inside a stream
 *     capture a call that would have to block returns BEAGLE_ERR_NOT_RESERVED and enqueues nothing.
 *   - Argument errors are returned synchronously and nothing is enqueued.
 *   - Data-dependent problems are reported in band: a malformed individual gets the canonical
 *     quiet NaN 0x7FC00000 as its fitness and never causes an out-of-bounds access.
 *   - Lower fitness is better for beagle_eval (MSE); the score-type fitness functions of beagle_eval_fit are
 *     maximised. A non-finite fitness marks an invalid individual.
 *   - One call at a time per process, on one device (the workspace is shared and belongs to the device that was
 *     current at the first call); calls are not re-entrant. The fitness function is an argument, never state.
 */
#ifndef BEAGLE_H_
#define BEAGLE_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- genome encoding (R2; north_star: "postfix int32 tokens {opcode:8, arg:24}") ----
 * A token is a 32-bit word read as unsigned: opcode = w & 0xFF, arg = w >> 8 (24 bits).
 * Opcode 0 is invalid on purpose so that zeroed memory is a malformed program.                  */
#define BEAGLE_OP_CONST 0x01 /* push consts[arg], arg < n_consts */
#define BEAGLE_OP_LOAD  0x02 /* push X[i][arg], arg < d */
#define BEAGLE_OP_ADD   0x03 /* a b -> a + b     */
#define BEAGLE_OP_SUB   0x04 /* a b -> a - b  (second-top minus top)     */
#define BEAGLE_OP_MUL   0x05 /* a b -> a * b     */
#define BEAGLE_OP_DIV   0x06 /* a b -> |b| < 1e-6f ? 1 : a / b  (protected) PAPER.md:238     */
#define BEAGLE_OP_SIN   0x07 /* a -> sin a     */
#define BEAGLE_OP_COS   0x08 /* a -> cos a     */
#define BEAGLE_OP_LOG   0x09 /* a -> |a| < 1e-6f ? 0 : ln|a|    (protected) PAPER.md:253     */
#define BEAGLE_OP_SQRT  0x0A /* a -> sqrt|a|                    (protected) PAPER.md:249     */
#define BEAGLE_OP_EXP   0x0B /* a -> exp(a > 80 ? 80 : a)       (clamped)     */
/* The rest of Table 3 in its own order from 0x10. DUP SWAP DEL SIGN SQUARE CUBE are compiled to
 * micro-ops and run on the interpreter like the eleven commands above (the stack commands are resolved at compile
 * time on terminals and cost a slot move on computed values). An individual that uses POW, one of the six library
 * functions or COPY / PASTE is evaluated by the blockwise kernel inside the same call (same definition, same
 * summation order, bit-identical where both apply, lower throughput).                                           */
#define BEAGLE_OP_DUP    0x10 /* a -> a a     */
#define BEAGLE_OP_SWAP   0x11 /* a b -> b a     */
#define BEAGLE_OP_DEL    0x12 /* a ->     */
#define BEAGLE_OP_SIGN   0x14 /* a -> -a     */
#define BEAGLE_OP_SQUARE 0x15 /* a -> a * a     */
#define BEAGLE_OP_CUBE   0x16 /* a -> (a * a) * a     */
#define BEAGLE_OP_CBRT   0x17 /* a -> cbrt a     */
#define BEAGLE_OP_TAN    0x18 /* a -> tan a     */
#define BEAGLE_OP_ARCSIN 0x19 /* a -> asin a   (NaN outside [-1, 1])     */
#define BEAGLE_OP_ARCCOS 0x1A /* a -> acos a   (NaN outside [-1, 1])     */
#define BEAGLE_OP_ARCTAN 0x1B /* a -> atan a     */
#define BEAGLE_OP_TANH   0x1C /* a -> tanh a     */
#define BEAGLE_OP_POW    0x13 /* a b -> pow(a, b)  (the C function)     */
#define BEAGLE_OP_COPY   0x1D /* variable @arg = top; stack unchanged     */
#define BEAGLE_OP_PASTE  0x1E /* push variable @arg; the variable is gone     */
#define BEAGLE_MAX_VARS  32   /* variable identifiers @0 .. @31; COPY and PASTE come in pairs: PASTE of a variable
                                 that holds nothing, COPY to one that does, or a COPY left without its PASTE make
                                 the program malformed                                                        */
#define BEAGLE_TOKEN(op, arg) ((int32_t)(((uint32_t)(arg) << 8) | ((uint32_t)(op) & 0xFFu)))

/* ---- limits (also returned by beagle_limits) ---- */
#define BEAGLE_MAX_LEN   512  /* tokens per individual (config 5 of BASELINE.json: 1..512)      */
#define BEAGLE_MAX_STACK 32   /* operand stack entries                            */
#define BEAGLE_MAX_N     1024 /* fitness cases per call                            */
#define BEAGLE_MAX_D     32   /* input variables per case                                       */
#define BEAGLE_MAX_CONSTS (1 << 24)

typedef int32_t beagle_status;
enum {
    BEAGLE_OK = 0,
    BEAGLE_ERR_INVALID_ARG = -1, /* null pointer with P > 0, size out of range                   */
    BEAGLE_ERR_UNSUPPORTED = -2, /* device is not sm_100, or not enough shared memory            */
    BEAGLE_ERR_CUDA = -3,        /* a CUDA call failed; see beagle_last_cuda_error               */
    BEAGLE_ERR_NOMEM = -4,       /* workspace or staging allocation failed                       */
    BEAGLE_ERR_NOT_RESERVED = -5 /* the call would have to block (grow its workspace) inside a
                                    stream capture; nothing was enqueued: beagle_reserve first    */
};

/* beagle_eval — score a device-resident colony.
 *
 * For every individual p in [0,P): run its postfix program on each of the N fitness cases
 * (Table 3 semantics with the protected forms above, fp32), take out_i = top of stack, and return
 *     fitness_out[p] = (sum_i (out_i - y[i])^2) / N + tax * lengths[p]          (D5)
 * in input order. The sum is taken before the division; the fp32 summation order is fixed (bitwise
 * reproducible run to run, independent of P, of the order of individuals and of chunking).
 *
 *   genomes      DEVICE  packed tokens, T = sum(lengths) words, 4-byte aligned; individual p owns
 *                        [off[p], off[p] + lengths[p]) with off = exclusive prefix sum of lengths
 *   lengths      DEVICE  P entries; an entry outside [1, BEAGLE_MAX_LEN] marks the individual
 *                        malformed and counts as 0 words in the prefix sum
 *   P            number of individuals, >= 0; P == 0 returns BEAGLE_OK and enqueues nothing
 *   consts       DEVICE  fp32 side table of n_consts entries; may be NULL iff n_consts == 0
 *   n_consts     0 .. BEAGLE_MAX_CONSTS
 *   X            DEVICE  N x d row-major fp32 (case-major)
 *   y            DEVICE  N fp32 targets
 *   N, d         1..BEAGLE_MAX_N, 1..BEAGLE_MAX_D
 *   tax          length tax per token (in north_star's float form)
 *   fitness_out  DEVICE  P fp32
 *   stream       cudaStream_t
 *
 * Device resources: the interpreter kernel takes all 512 tensor-memory columns and up to 227 KB of shared
 * memory of every SM for the duration of the call (one CTA per SM). When the fitness cases do not fit tensor
 * memory (d > 16 at N > 512; d <= 32 always fits at N <= 512) the call runs the blockwise kernel instead: same
 * result bit for bit, lower throughput.
 *
 * Malformed (fitness = quiet NaN 0x7FC00000): length outside [1,512], an opcode outside the table above, non-zero
 * arg on an operator, CONST arg >= n_consts, LOAD arg >= d, a command that needs more entries than the
 * stack holds, depth above 32, an empty stack at the end (DEL can empty it in between).
 * The extent of `genomes` is trusted to be sum of the in-range lengths.                          */
beagle_status beagle_eval(const int32_t* genomes, const int32_t* lengths, int64_t P,
                          const float* consts, int64_t n_consts,
                          const float* X, const float* y, int32_t N, int32_t d,
                          float tax, float* fitness_out, void* stream);

/* beagle_eval_fit — the same path with the fitness function chosen by `fit`.
 *
 *   BEAGLE_FIT_MSE          fitness = MSE + tax * L (beagle_eval; M is ignored)
 *   BEAGLE_FIT_CORRELATION  the paper's default objective (Eq. 1-2; Eq. 3-4 at P:494-501):
 *                           a case is a valid pair when the model output and the target are both finite;
 *                           c1 = pairs with exactly one side finite, c2 = pairs with neither;
 *                           r = Pearson correlation over the valid pairs (means over the valid pairs);
 *                           score = M r^4 (N - (c1 + c2)) - M (c1 - c2);  fitness = score - tax * L, MAXIMISED.
 *                           r = 0 when fewer than two valid pairs are left or either side has zero variance
 *                           there (R23). y may hold NaN / Inf. A well-formed program always gets a
 *                           finite-or-NaN float; malformed programs get the canonical quiet NaN as in beagle_eval.
 *   BEAGLE_FIT_STD, _SQUARE, _CUBE, _HYPER   the point-to-point integer-reward family (Eq. 5 at
 *                           P:503-506), p = 1, 2, 3, 8: per valid pair  M  if max(|f|,|y|) = 0, else
 *                           round(M q^p - [f, y of opposite sign] M/11), q = min(|f|,|y|) / max(|f|,|y|), computed in
 *                           fp32, round half to even; a pair with one side finite scores -M, with neither +M;
 *                           fitness = sum over the cases - tax * L, MAXIMISED (D9, R25). Exact (integers) while
 *                           M * N < 2^24.
 *   M                       the maximum score per case (BConfig.MaxScore; the paper's logs imply 10000)
 *
 * All other arguments, limits and errors as beagle_eval; an unknown `fit` returns BEAGLE_ERR_INVALID_ARG.       */
#define BEAGLE_FIT_MSE         0
#define BEAGLE_FIT_CORRELATION 1
#define BEAGLE_FIT_STD         2   /* StdFitFunc        (Eq. 5)                       */
#define BEAGLE_FIT_STD_SQUARE  3   /* StdSquareFitFunc: the ratio of Eq. 5 squared    */
#define BEAGLE_FIT_STD_CUBE    4   /* StdCubeFitFunc:   ... cubed                     */
#define BEAGLE_FIT_STD_HYPER   5   /* StdHyperFitFunc:  ... to the power 8            */
beagle_status beagle_eval_fit(const int32_t* genomes, const int32_t* lengths, int64_t P,
                              const float* consts, int64_t n_consts,
                              const float* X, const float* y, int32_t N, int32_t d,
                              int32_t fit, float M, float tax, float* fitness_out, void* stream);

/* beagle_eval_chunked — the same result for a colony held in HOST memory that may be larger than
 * the device budget ("manages populations in batches to ensure the GPU memory is
 * never exceeded"; R19). The colony is cut at individual boundaries into chunks of at
 * most device_budget_bytes/K bytes of tokens+lengths, K = device_budget_bytes / 32 MiB clamped to 2..8 staging
 * buffers (beagle_set_chunk_target changes the 32 MiB); chunk c goes to buffer c mod K, and the chunks after chunk c
 * are copied host-to-device on an internal copy stream while chunk c is evaluated on `stream`.
 * fitness_out is bit-identical to beagle_eval on the whole colony, for any budget.
 *
 *   h_genomes, h_lengths, h_consts   HOST (pinned memory for overlap; pageable memory works but
 *                                    the copies then do not overlap)
 *   X, y, fitness_out                DEVICE, as in beagle_eval
 *   device_budget_bytes              cap on device bytes used for genome staging (all K buffers together);
 *                                    every buffer must hold one maximum-length individual: at least
 *                                    2 * 4 * (BEAGLE_MAX_LEN + 64) = 4608 bytes, else BEAGLE_ERR_INVALID_ARG
 * The first call with a new budget allocates the staging buffers (blocking; beagle_reserve_chunked does it ahead).
 * Completion of `stream` implies completion of everything, copies included. The host arrays must
 * stay valid and unchanged until then.                                                           */
beagle_status beagle_eval_chunked(const int32_t* h_genomes, const int32_t* h_lengths, int64_t P,
                                  const float* h_consts, int64_t n_consts,
                                  const float* X, const float* y, int32_t N, int32_t d,
                                  float tax, float* fitness_out,
                                  int64_t device_budget_bytes, void* stream);

/* beagle_eval_chunked_fit — beagle_eval_chunked with the fitness function of beagle_eval_fit (`fit`, `M` as there);
 * bit-identical to beagle_eval_fit on the whole colony, for any budget.                                          */
beagle_status beagle_eval_chunked_fit(const int32_t* h_genomes, const int32_t* h_lengths, int64_t P,
                                      const float* h_consts, int64_t n_consts,
                                      const float* X, const float* y, int32_t N, int32_t d,
                                      int32_t fit, float M, float tax, float* fitness_out,
                                      int64_t device_budget_bytes, void* stream);

/* beagle_rank — Monte-Carlo ranking, the step that follows scoring:
 * "Beagle takes a random sample of 100 individuals and uses those 100 individuals to estimate the population
 * percentiles. Through one pass of the population then, individuals are assigned to their specific percentile and are
 * given rank proportional breeding rights" (Table 2). The random draw is the caller's, so the call is deterministic.
 *
 *   fitness      DEVICE  P fp32, as written by beagle_eval / beagle_eval_fit (stays on the device: no D2H of P floats)
 *   sample_idx   DEVICE  n_sample int64 indices into fitness, each in [0, P)  (trusted; the paper draws 100)
 *   n_sample     1 .. 1024
 *   maximise     0: lower fitness is better (MSE); non-zero: higher is better (correlation score)
 *   decile_out   DEVICE  P bytes: g = min(9, 10 * worse / n_sample), worse = number of sampled individuals strictly
 *                        worse than this one; group g is Table 2's row "percentile >= 10 g". A NaN fitness is worse
 *                        than every number; equal fitnesses are not strictly worse (R24).
 *   hist_out     DEVICE  10 int64: individuals per group (zeroed by the call); may be NULL
 *
 * BEAGLE_TABLE2[g] = expected number of children of group g (Table 2): expected births of the next
 * generation = sum over g of hist_out[g] * BEAGLE_TABLE2[g].                                                    */
static const float BEAGLE_TABLE2[10] = { 0.01f, 0.03f, 0.06f, 0.15f, 0.25f, 0.5f, 1.0f, 1.5f, 2.5f, 4.0f };
beagle_status beagle_rank(const float* fitness, int64_t P, const int64_t* sample_idx, int32_t n_sample,
                          int32_t maximise, uint8_t* decile_out, int64_t* hist_out, void* stream);

/* beagle_eval_blockwise — prior art kept as a measured baseline, not the product: the paper's own
 * mapping (one CUDA block per individual, one thread per fitness case, a 32-entry
 * per-thread stack in local memory, block aggregation in shared memory), same arguments and the
 * same definition of the result as beagle_eval, the same per-command functions and the same
 * summation order: its results are bit-identical to beagle_eval's (tests/test_gpu_edges.py). It
 * is also the kernel that takes, inside beagle_eval, the individuals the interpreter cannot.    */
beagle_status beagle_eval_blockwise(const int32_t* genomes, const int32_t* lengths, int64_t P,
                                    const float* consts, int64_t n_consts,
                                    const float* X, const float* y, int32_t N, int32_t d,
                                    float tax, float* fitness_out, void* stream);

/* beagle_debug_outputs — test only: per-case program outputs, out_PxN[p*N + i] (DEVICE, P*N fp32),
 * computed by the same interpreter as beagle_eval; malformed individuals give NaN rows.          */
beagle_status beagle_debug_outputs(const int32_t* genomes, const int32_t* lengths, int64_t P,
                                   const float* consts, int64_t n_consts,
                                   const float* X, int32_t N, int32_t d,
                                   float* out_PxN, void* stream);

/* beagle_debug_schedule — test only: copies what the scheduling pre-pass (offsets, per-program
 * scan, length-sorted permutation) produced for the last beagle_eval/debug call on `stream`.
 * Any pointer may be NULL. DEVICE outputs: off[P] (int64 exclusive prefix sum), depth[P] (int32
 * maximum stack depth, 0 if malformed), perm[P] (int32, the evaluation order: the individuals with a
 * length in [1, 512] sorted by length, longest first, then -1 for the others). Enqueued on `stream`. */
beagle_status beagle_debug_schedule(int64_t P, int64_t* off, int32_t* depth, int32_t* perm,
                                    void* stream);

/* beagle_debug_counts — test only: what the pre-pass of the last beagle_eval / debug call on `stream` (for a chunked
 * call: of its last chunk) counted. HOST outputs, any may be NULL; synchronises `stream`. n_sorted: individuals with a
 * length in [1, 512]; n_general: of those, the ones that are not trees of the eleven hot-path commands (compiled by
 * k_compile_general); n_slow: individuals handed to the blockwise kernel (POW, library functions, COPY / PASTE, or no
 * room in the workspace); n_malformed: in-range individuals that are not programs (D3).               */
beagle_status beagle_debug_counts(int32_t* n_sorted, int32_t* n_general, int32_t* n_slow, int32_t* n_malformed, void* stream);

/* beagle_debug_plan — test only, HOST only, needs no device: the plan of tensor memory and shared memory (DESIGN.md section 7,
 * "the plan of the 32 TMEM rows") that a call with N cases, d variables, fitness function `fit` (BEAGLE_FIT_*) and, for
 * fitness_only != 0, no per-case outputs would get on a device with smem_optin bytes of opt-in shared memory per block.
 * out12 (HOST): 0 fast (the interpreter takes the call; 0: the blockwise kernel), 1 split (one launch per pass of 512 cases),
 * 2 threads per block, 3 variable rows, 4 reciprocal rows, 5 slot rows per warp, 6 variables with staged unary rows,
 * 7 bytes of a warp's record ring, 8 dynamic shared memory in bytes, 9-11 byte offsets of y, the unary rows, the rings.
 * BEAGLE_ERR_INVALID_ARG for arguments out of range. */
beagle_status beagle_debug_plan(int32_t N, int32_t d, int32_t fit, int32_t fitness_only, int32_t smem_optin, int32_t* out12);

/* beagle_debug_chunk_plan — test only, HOST only, needs no device: the chunks beagle_eval_chunked would cut a colony with these
 * HOST lengths into under this budget (the same code: the budget cut into K buffers, beagle_set_chunk_target; a chunk = as many
 * whole individuals as fit one buffer at one word per individual plus one per token, three words spare). ends[i] (HOST, up to
 * max_ends entries, may be NULL) = the index after the last individual of chunk i; *n_chunks, *n_buffers (K), *buffer_bytes: any may
 * be NULL. BEAGLE_ERR_INVALID_ARG as beagle_eval_chunked for the same arguments. */
beagle_status beagle_debug_chunk_plan(const int32_t* h_lengths, int64_t P, int64_t device_budget_bytes, int64_t* ends, int64_t max_ends,
                                      int64_t* n_chunks, int32_t* n_buffers, int64_t* buffer_bytes);

/* beagle_debug_walk_tables — test only, HOST only: the two tables that drive the tree compiler's walk, as the device gets them:
 * lut160 = 10 rows (nothing; SIN COS LOG SQRT EXP; ADD SUB MUL DIV) of 16 entries indexed by what the two topmost stack entries
 * are (a computed? b computed? a a variable? b a variable?), tok130 = 65 pairs of words per opcode byte (64: past the end of the
 * program). Either may be NULL. Field layout: compile_kernel.inc. */
void beagle_debug_walk_tables(uint32_t* lut160, uint32_t* tok130);

/* beagle_debug_compile — test only, HOST only, needs no device: the compiler of the whole language (the function k_compile_general runs
 * one lane per program on the device, compiled for the host as well) on ONE program. tokens: HOST, len words (1..512); consts: HOST;
 * tmem_slots, k_rcp, k_un, un_row_bytes: the plan the records are compiled for (beagle_debug_plan: slot rows per warp, variables with
 * a reciprocal row, variables with staged unary rows, bytes per staged row); rcp_unsafe: bit j set = variable j has a case with
 * |x| < 1e-6f (its division is protected: no reciprocal row). Outputs (HOST): *depth = the maximum stack depth, 0 if the program is
 * malformed (D3); *slow = 1 if it is handed to the blockwise kernel (POW, a library function, COPY / PASTE); otherwise
 * records[2 i], records[2 i + 1] = the words h, o of micro-op i (csrc/uop.cuh; room for len + 1 records) and *n_records their number,
 * before the END record. One difference from the device: the reciprocal a constant divisor is folded to is the IEEE 1 / c here,
 * the division handler's rcp.approx there. BEAGLE_ERR_INVALID_ARG for arguments out of range. */
beagle_status beagle_debug_compile(const int32_t* tokens, int32_t len, const float* consts, int64_t n_consts, int32_t d,
                                   int32_t tmem_slots, int32_t k_rcp, int32_t k_un, int32_t un_row_bytes, uint32_t rcp_unsafe,
                                   uint32_t* records, int32_t* n_records, int32_t* depth, int32_t* slow);

/* (The three calls below run on the SIMT emulator, which needs up to 1024 OS threads at a time: BEAGLE_ERR_UNSUPPORTED if the host refuses them.) */
/* beagle_debug_corr — test only, HOST only, needs no device: the correlation fitness (BEAGLE_FIT_CORRELATION) of ONE individual from its
 * per-case outputs f[0..N) and the targets y[0..N) (HOST), by the device's own reduction (csrc/fit_corr.cuh compiled for the host: IEEE
 * single precision throughout, so the device's bits) on one warp of the SIMT emulator, in the kernels' layout of 16 cases per lane and
 * pass. len, M, tax as in beagle_eval_fit. pre != 0: full passes with finite targets take the version with the target's side computed
 * once (the interpreter kernel's way), else the general one (the blockwise kernel's way); the two give the same bits. */
beagle_status beagle_debug_corr(const float* f, const float* y, int32_t N, int32_t len, float M, float tax, int32_t pre, float* fitness_out);

/* beagle_debug_rank — test only, HOST only, needs no device: k_rank (csrc/rank_body.inc, the source the kernel is compiled from) run on HOST
 * memory by the SIMT emulator, `grid` blocks of 256 threads one after the other (beagle_rank launches up to 8 per SM). Arguments as
 * beagle_rank with HOST pointers; sample_idx is checked here (each in [0, P)); hist_out is required. 1 <= P <= 2^22. */
beagle_status beagle_debug_rank(const float* fitness, int64_t P, const int64_t* sample_idx, int32_t n_sample, int32_t maximise,
                                int32_t grid, uint8_t* decile_out, int64_t* hist_out);

/* beagle_debug_prepass — test only, HOST only, needs no device: the scheduling pre-pass (k_len_pass1, k_len_pass2, k_scatter: offsets, the
 * length histogram and its scans, the counting sort by length, the start records, the transpose of the cases; csrc/prepass_body.inc, the
 * source the three kernels are compiled from) run on HOST memory by a small SIMT emulator (one OS thread per CUDA thread of a block,
 * csrc/simt_host.inc), with the launch shapes of the real call. lengths: P entries (1 <= P <= 2^24); X, y as beagle_eval but HOST; split:
 * the layout flag of a call split by passes. Outputs (HOST): off[P] (exclusive prefix sum of the in-range lengths), sched4[4 P] (the start
 * record of each sorted position: individual, token offset (low 32 bits), record base (low 32 bits), length | high bits; positions past
 * n_sorted are not written), fitness[P] and depth[P] (written for out-of-range lengths only: quiet NaN and 0), xt[(d + 1) * npad] (the
 * cases variable-major, zero-padded to a multiple of 512, y as row d), hdr6 = { T, micro-op entries reserved, n_sorted, max_len, mask of
 * variables with a protected case, 0 (-1: the length histogram was not left zeroed for the next call) }, binstart[513], binubase[513]. */
beagle_status beagle_debug_prepass(const int32_t* lengths, int64_t P, const float* X, const float* y, int32_t N, int32_t d, int32_t split,
                                   int64_t* off, int32_t* sched4, float* fitness, int32_t* depth, float* xt, int64_t* hdr6,
                                   int32_t* binstart, int64_t* binubase);

/* beagle_debug_queue — test only, HOST only, needs no device: the scheduling loop of ONE warp of the interpreter kernel (csrc/queue_body.inc,
 * the source both k_eval and this call are compiled from) over a given queue. meta4: HOST, `total` entries of four ints as k_compile leaves
 * them in evaluation order (x = individual, y = record block in 16-byte units, z = records to copy, 0 = nothing to run, w = length);
 * max_len, ring_bytes, grid, threads: what the launch would have (longest program, bytes of a warp's ring, CTAs, threads per CTA);
 * grouped != 0: the MSE-without-outputs instantiation (one interpreter entry per group). skip_seed != 0: after each visit of this warp the
 * queue moves on by 0..3 more batches (other warps' visits); queue_start: where the queue stands when the warp arrives.
 * events (HOST, cap x 4 ints; *n_events = how many there were): 0 visit (first entry, batch); 1 bulk copy (stage, source in 16-byte units,
 * bytes); 2 barrier wait (stage, phase parity); 3 a group handed to the interpreter (byte offset in the ring, programs); 4 one program
 * handed to it (byte offset, individual, length). sizing3: entries per visit, bytes per stage, stages. */
beagle_status beagle_debug_queue(const int32_t* meta4, int32_t total, int32_t max_len, int32_t ring_bytes, int32_t grid, int32_t threads,
                                 int32_t grouped, uint32_t skip_seed, uint32_t queue_start, int32_t* events, int32_t cap,
                                 int32_t* n_events, int32_t* sizing3);

/* beagle_debug_walk — test only, HOST only, needs no device: the body of k_compile's table-driven walk (csrc/walk_body.inc, the source
 * both the kernel and this call are compiled from) on ONE program; f1 != 0: the instantiation that also takes DUP SWAP DEL SIGN SQUARE
 * CUBE (f1 == 2: with the warp-wide vote that guards those commands passed at every token, as for a lane whose neighbours meet them; bits 17:8 of f1: the
 * walk goes on for that many tokens past the program's end, as for a lane beside a longer program of its warp). Arguments as beagle_debug_compile. *taken = 1 if the walk compiled the program, 0 if it turned it down (anything that is not
 * a well-formed program of its commands: k_compile_general looks at those); for taken programs *depth, records and *n_records as
 * beagle_debug_compile, *used_f1 = 1 if one of the six extra commands occurred. Same difference from the device (1 / c in IEEE). */
beagle_status beagle_debug_walk(const int32_t* tokens, int32_t len, const float* consts, int64_t n_consts, int32_t d,
                                int32_t tmem_slots, int32_t k_rcp, int32_t k_un, int32_t un_row_bytes, uint32_t rcp_unsafe, int32_t f1,
                                uint32_t* records, int32_t* n_records, int32_t* depth, int32_t* taken, int32_t* used_f1);

/* beagle_debug_std_reward — test only, HOST only, needs no device: the reward of each (f[i], y[i]) pair under the Std family
 * (BEAGLE_FIT_STD, _SQUARE, _CUBE, _HYPER; Eq. 5), computed by the device's own function compiled for the host (the integer is decided
 * in fp32: the same IEEE operations in the same order on both). f, y, out: HOST, n floats. BEAGLE_ERR_INVALID_ARG for another `fit`. */
beagle_status beagle_debug_std_reward(const float* f, const float* y, int64_t n, int32_t fit, float M, float* out);

/* Limits compiled into the library (any pointer may be NULL). */
void beagle_limits(int32_t* max_len, int32_t* max_stack, int32_t* max_n, int32_t* max_d);

/* Static, NUL-terminated description of a status code. */
const char* beagle_status_string(beagle_status s);

/* The cudaError_t behind the most recent BEAGLE_ERR_CUDA / BEAGLE_ERR_NOMEM (0 if none). */
int32_t beagle_last_cuda_error(void);

/* Pre-size the workspace for colonies of up to P_max individuals and T_max tokens so that later
 * calls with P <= P_max and at most T_max tokens never block (see "Blocking" above). T_max = 0 sizes the
 * per-individual arrays only. Synchronises the device if it has to reallocate. Individuals of a call that breaks
 * the promise (more tokens than T_max) and do not fit are evaluated by the blockwise kernel: same results. */
beagle_status beagle_reserve(int64_t P_max, int64_t T_max);

/* Pre-size the staging buffers of beagle_eval_chunked for this budget. */
beagle_status beagle_reserve_chunked(int64_t device_budget_bytes);

/* Free the cached workspace and staging buffers (synchronises the device). */
void beagle_release(void);

/* Number of kernels the most recent beagle_eval* call launched (for bench.py's gpu_launches). */
int32_t beagle_last_launch_count(void);

/* Size the staging buffers of beagle_eval_chunked aim at (default 32 MiB; bytes <= 0 restores it): the budget is
 * cut into K = budget / target buffers, 2 <= K <= 8. beagle_chunk_buffers returns the K in use (0: none yet). */
void    beagle_set_chunk_target(int64_t bytes);
int32_t beagle_chunk_buffers(void);

/* Profiling hooks for bench.py's roofline line. While profiling is on (on = n > 0), every n-th beagle_eval
 * call, starting with the first, brackets its pre-pass and its evaluation kernels (the interpreter launches) with
 * three CUDA events on `stream` (at most 256 calls are recorded; later ones are not). The two
 * event records cost a call about 12 us of stream bubbles and keep k_eval from starting under the tail of
 * k_compile, which is why a bench may want n > 1.
 * beagle_profiled_eval_kernel_ms synchronises on the recorded events, stores the number of
 * recorded calls in *n_calls (may be NULL) and returns their mean device time in milliseconds
 * (< 0 if nothing was recorded). beagle_set_profiling(1) clears the record. */
void  beagle_set_profiling(int32_t on);
float beagle_profiled_eval_kernel_ms(int32_t* n_calls);
/* The same for the pre-pass of the recorded calls (a2-a3 and the compile step of a5: from the start of the call to
 * the start of the interpreter), mean device time in milliseconds. */
float beagle_profiled_prepass_ms(int32_t* n_calls);

#ifdef __cplusplus
}
#endif
#endif /* BEAGLE_H_ */

/* mfsdp.h -- C ABI of the owner-local optimizer step of MatrixFSDP (arxiv/paper_2607_05895), B200 / sm_100a.
 *
 * What the library computes (PAPER.md = /root/reference/PAPER.md, the paper text):
 *   PAPER.md:45   each DP-sharded 2D weight lives whole on one owner rank; the non-2D tensors of an FSDP unit
 *                 are packed into one tail role on a tail owner and stay on AdamW.
 *   PAPER.md:47   "The owner applies the Newton-Schulz update to the full matrix and updates its local parameter
 *                 and Muon state, so the optimizer step contains no matrix all-gather, broadcast, or
 *                 redistribute.  Tail owners apply AdamW to their packed non-matrix tensors."
 *   PAPER.md:97   optimizer routing: Muon sees a matrix only on its owner, tail-owner shards go to AdamW.
 *   PAPER.md:101-107 (Algorithm 1) + PAPER.md:65-71: the balance-aware owner planner.
 * The Muon arithmetic itself (the paper never prints it) is fixed by BASELINE.json's north_star and the readings
 * listed in DESIGN.md section 4: EMA Nesterov momentum, Frobenius normalisation with eps clamp, K-step quintic
 * Newton-Schulz (A = X X^T, B = bA + cA^2, X <- aX + BX, tall matrices transposed), scaled decoupled-decay update.
 *
 * Conventions
 *   * Plain C, POD structs with fixed-width fields, no torch / C++ types.  Every pointer is annotated HOST or DEVICE.
 *   * Ownership: the caller owns every buffer.  The library never allocates or frees caller-visible device memory
 *     and keeps no state except a small per-process cache of host-built launch tables (tensor maps, tile tables).
 *   * Asynchrony: the *_step functions enqueue work on `cuda_stream` (a cudaStream_t passed as void*, NULL = the
 *     legacy default stream) and return without synchronising.  G is read-only; W, M (P, m, v) are updated in place.
 *   * Errors: 0 on success, a negative MFSDP_E* code otherwise; nothing is printed, nothing throws or aborts.
 *   * Determinism: same inputs give bit-identical outputs, run to run.  The Newton-Schulz tiles are handed to the
 *     SMs by a DYNAMIC scheduler (an atomic claim counter), so which unit computes a tile and when varies; every
 *     output tile is computed by exactly one unit with a fixed k order, and every norm by a fixed-order reduction,
 *     so the values do not depend on the schedule (tests/test_gpu_parity.py::test_run_to_run_determinism).
 *   * Dynamic range: the Frobenius normalisation is folded into the first Newton-Schulz iteration (the Gram matrix
 *     of the UNNORMALISED bf16/fp32 momentum update U is accumulated in fp32 and scaled by 1/||U||^2 afterwards), so
 *     u_i u_j must stay inside fp32's normal range: supported rms(U) is about 1e-17 .. 1e+16 (gradients of real
 *     training runs sit around 1e-6 .. 1e+2).  Inside that range, and above the clamp ||U||_F >= eps, the result is
 *     invariant to the scale of G exactly like the definition (power-of-two scalings give bit-identical O; tested);
 *     below eps the clamp X0 = U / eps applies, as in the definition.
 *   * There is NO CPU fallback: on a machine without an sm_100 device the step functions return MFSDP_EARCH.
 */
#ifndef MFSDP_H_
#define MFSDP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- enums (plain ints in the ABI) ------------------------------------------------------------------------- */
enum { MFSDP_BF16 = 0, MFSDP_F32 = 1 };                       /* storage dtype of W / G (tails: P / G)            */
enum { MFSDP_ROLE_MATRIX = 0, MFSDP_ROLE_TAIL = 1 };          /* PAPER.md:103 Alg. 1 line 1                       */
enum { MFSDP_POLICY_ROLE_GREEDY = 0,                          /* PAPER.md:104 Alg. 1 line 2                       */
       MFSDP_POLICY_SCOPE_GREEDY = 1,                         /* PAPER.md:105 Alg. 1 line 3                       */
       MFSDP_POLICY_COST_AWARE = 2 };                         /* PAPER.md:106 Alg. 1 line 4 (mfsdp_plan_ex)       */
enum { MFSDP_METRIC_NUMEL = 0,                                /* PAPER.md:65 "greedy load is owner-resident numel" */
       MFSDP_METRIC_NS_FLOPS = 1 };                           /* BASELINE.json C4/C5: m^2 (2n + m), m=min n=max    */
enum { MFSDP_SCALE_MATCH_RMS_ADAMW = 0,                       /* 0.2 sqrt(max(rows, cols))       */
       MFSDP_SCALE_ORIGINAL = 1,                              /* sqrt(max(1, rows / cols))                        */
       MFSDP_SCALE_NONE = 2 };
enum { MFSDP_NS_BF16 = 0,                                     /* bf16 operands, fp32 accumulate (tcgen05)         */
       MFSDP_NS_FP32 = 1 };                                   /* fp32 operands and accumulate (FFMA), no TF32     */
enum { MFSDP_PARAM_SKIP = 1u };                               /* mfsdp_param_t.flags bit0 (PAPER.md:45 TP skip)   */
enum { MFSDP_DESC_TRANSPOSED = 1u };                          /* mfsdp_desc_t.flags bit0: rows > cols (NS runs on X^T) */
enum { MFSDP_STEP_KEEP_O = 1u };                              /* mfsdp_muon_hparams_t.flags bit0: mfsdp_muon_step also
                                                                 leaves O = X_K in the workspace (see mfsdp_muon_step) */
enum { MFSDP_SEG_ALIGN = 64 };                                /* every segment starts on a 64-element boundary    */

enum { MFSDP_OK = 0, MFSDP_EINVAL = -1, MFSDP_ECAP = -2, MFSDP_ELAYOUT = -3, MFSDP_EARCH = -4, MFSDP_ECUDA = -5,
       MFSDP_ECACHE = -6,                                     /* launch-table cache full, see mfsdp_release_plans  */
       MFSDP_ETOOBIG = -7 };                                  /* matrix beyond the fixed scratch of mfsdp_momentum_pass_static */

/* ---- records ------------------------------------------------------------------------------------------------ */
/* One model parameter, in model order (planner input). */
typedef struct {
  uint32_t block_id; /* FSDP unit; non-decreasing in model order                                                  */
  uint32_t ndim;     /* 2 -> matrix role; anything else -> member of the block's tail role                        */
  uint32_t rows;     /* ndim != 2: rows = numel, cols = 1                                                         */
  uint32_t cols;
  uint32_t dtype;    /* MFSDP_BF16 | MFSDP_F32                                                                    */
  uint32_t flags;    /* MFSDP_PARAM_SKIP                                                                          */
} mfsdp_param_t;

/* One resident segment of one rank (planner output, step input): the analogue of the paper's MatrixShard layout
 * entry: "one full segment per 2D matrix, one packed tail segment per block".
 * Matrices live in one rank-flat element space (W, G, M share offsets), tails in another (P, G, m, v). */
typedef struct {
  uint32_t role;     /* MFSDP_ROLE_MATRIX | MFSDP_ROLE_TAIL                                                       */
  uint32_t param_id; /* index into params[] (a tail: index of its first member)                                   */
  uint32_t block_id;
  uint32_t rows;     /* as stored, row-major, cols contiguous.  tail: rows = packed numel, cols = 1               */
  uint32_t cols;
  uint32_t dtype;
  uint32_t flags;    /* MFSDP_DESC_TRANSPOSED                                                                     */
  uint32_t reserved; /* 0                                                                                         */
  uint64_t elem_off; /* offset in ELEMENTS into the rank-flat buffers of its element space; multiple of 64        */
} mfsdp_desc_t;

/* Hyper-parameters are doubles so that derived constants (1 - mu, 1 - lr wd, 1 - beta^t) are formed in double on
 * the host and rounded once to the kernels' fp32. */
typedef struct {
  double  lr;            /* eta                                                                                   */
  double  weight_decay;  /* lambda, decoupled: W <- W (1 - eta lambda) - eta s O                                  */
  double  momentum;      /* mu: M <- mu M + (1 - mu) G                                                            */
  double  a, b, c;       /* quintic coefficients (north_star fallback 3.4445, -4.7750, 2.0315)                    */
  double  eps;           /* X0 = U / max(||U||_F, eps), 1e-7                                                      */
  int32_t nesterov;      /* != 0: U = (1 - mu) G + mu M ; 0: U = M                                                */
  int32_t ns_steps;      /* K >= 1 (north_star: 5; the paper's runs: 2)                             */
  int32_t scale_mode;    /* MFSDP_SCALE_*                                                                         */
  int32_t precision;     /* MFSDP_NS_BF16 | MFSDP_NS_FP32                                                         */
  uint32_t flags;        /* MFSDP_STEP_*                                                                          */
  uint32_t reserved;     /* 0                                                                                     */
} mfsdp_muon_hparams_t;

typedef struct {
  double  lr, beta1, beta2, eps, weight_decay;
  int64_t step;          /* 1-based step count t used for bias correction                                         */
} mfsdp_adamw_hparams_t;

/* ---- planner (HOST only, no CUDA) -----------------------------------------------------------------------------
 * Algorithm 1, lines 1-5.  Roles are built from params[] (line 1), assigned greedily
 * ("largest roles to the currently lightest ranks", ties: load desc, block asc, parameter index asc; lightest rank
 * ties -> lowest rank id), and the resident set of `rank` (rank < 0: the heaviest rank by primary load, ties ->
 * lowest id) is emitted as a descriptor table in (block, parameter) order and validated (line 5: one contiguous,
 * aligned, non-overlapping segment per resident parameter).
 *   params, n_params    HOST in.   model parameters in model order.
 *   owner_out           HOST out.  [n_roles] owner rank per role, roles in model order; may be NULL.
 *   n_roles             HOST out.  number of roles; may be NULL.
 *   rank_load_out       HOST out.  [2 * world_size]: primary load vector then tail load vector (the latter is all
 *                                  zero under MFSDP_METRIC_NUMEL, where one vector carries both); may be NULL.
 *   desc_out, desc_cap  HOST out.  descriptor table of the chosen rank; desc_out == NULL -> size query only.
 *   n_desc              HOST out.  number of descriptors of the chosen rank (always written).
 *   rank_out            HOST out.  the rank actually chosen; may be NULL.
 * Returns MFSDP_EINVAL (null params with n_params > 0, world_size < 1, rank >= world_size, unknown policy/metric,
 * zero-sized parameter, decreasing block ids, tail members of one block with different dtypes), MFSDP_ECAP
 * (desc_cap < *n_desc; *n_desc holds the required count), MFSDP_ELAYOUT (validation failed). */
int mfsdp_plan(const mfsdp_param_t* params, size_t n_params, int world_size, int policy, int metric, int rank,
               int32_t* owner_out, size_t* n_roles, uint64_t* rank_load_out,
               mfsdp_desc_t* desc_out, size_t desc_cap, size_t* n_desc, int* rank_out);

/* Algorithm 1 line 4 ("COSTAWARE: use SCOPEGREEDY only if balance improves within workspace caps; else
 * use ROLEGREEDY").  The paper defines neither the caps nor the scorer; reading P5: the scope plan
 * is taken iff (a) its maximum primary load is strictly below the role plan's and (b), with O_{B,r} = bytes of block B
 * owned by rank r and ws[r] = the step-workspace estimate of mfsdp_score_plan,
 *   max_{B,r} O_{B,r}(scope) * owner_den <= owner_num * max_{B,r} O_{B,r}(role),
 *   max_r ws[r](scope) * ws_den <= ws_num * max_r ws[r](role),
 *   max_{B,r} O_{B,r}(scope) <= abs_owner_bytes and max_r ws[r](scope) <= abs_ws_bytes where those are non-zero. */
typedef struct {
  uint32_t owner_num, owner_den;     /* default 9 / 8 */
  uint32_t ws_num, ws_den;           /* default 9 / 8 */
  uint64_t abs_owner_bytes;          /* 0 = no absolute cap */
  uint64_t abs_ws_bytes;             /* 0 = no absolute cap */
} mfsdp_caps_t;

/* mfsdp_plan with the caps of MFSDP_POLICY_COST_AWARE (caps == NULL: the defaults; ignored by the other policies) and
 * the policy actually used (*policy_used, may be NULL: ROLE_GREEDY or SCOPE_GREEDY).  mfsdp_plan(policy = COST_AWARE)
 * is this call with caps == NULL.  MFSDP_EINVAL additionally for a zero denominator. */
int mfsdp_plan_ex(const mfsdp_param_t* params, size_t n_params, int world_size, int policy, int metric, int rank,
                  const mfsdp_caps_t* caps, int32_t* owner_out, size_t* n_roles, uint64_t* rank_load_out,
                  mfsdp_desc_t* desc_out, size_t desc_cap, size_t* n_desc, int* rank_out, int* policy_used);

/* Resource scorer ("expands a completed plan into per-rank parameter, gradient, optimizer-state,
 * communication, and workspace estimates") and the per-block bandwidth model of PAPER.md:77-81 (HOST, integers; the
 * formulas are DESIGN.md reading P5 -- the paper prints none):
 *   param_bytes[r]  sum over roles owned by r of numel * sizeof(dtype);   grad_bytes[r] = param_bytes[r];
 *   state_bytes[r]  4 * numel per owned matrix (fp32 Muon momentum) + 8 * numel per owned tail (AdamW m, v);
 *   comm_bytes[r]   sum over blocks of (W - 1) * O_{B,r}  (sent per materialisation pass = received per gradient
 *                   reduction pass; its per-block maximum over r is C_B^owner);
 *   workspace_bytes[r]  sum over owned matrices of 2 * (2 rows cols + 2 d^2): X ping-pong + A + P in bf16, unpadded
 *                   (mfsdp_workspace_bytes of the rank's table is this plus alignment padding and the norm scratch);
 *   max_block_owner_bytes[r] = max_B O_{B,r}: the largest owner segment r holds unsharded.
 * Per block B in model order: P_B, max_r O_{B,r}, gamma_B = max_r O_{B,r} / (P_B / W), C_B^FSDP = P_B (W-1)/W,
 * C_B^owner = (W-1) max_r O_{B,r} = gamma_B C_B^FSDP.
 *   owner, n_roles   HOST in.  owner rank per role as returned by mfsdp_plan (n_roles must match the roles of params).
 *   rank_out         HOST out. [world_size]; may be NULL.
 *   block_out, block_cap, n_blocks  HOST out. per-block records; block_out == NULL: only *n_blocks is written.
 * Returns MFSDP_EINVAL (bad params / owner out of range / n_roles mismatch), MFSDP_ECAP (block_cap too small). */
typedef struct {
  uint64_t param_bytes, grad_bytes, state_bytes, comm_bytes, workspace_bytes, max_block_owner_bytes;
} mfsdp_rank_score_t;
typedef struct {
  uint32_t block_id, reserved;
  uint64_t param_bytes;              /* P_B */
  uint64_t max_owner_bytes;          /* max_r O_{B,r} */
  double gamma, c_fsdp, c_owner;
} mfsdp_block_score_t;
int mfsdp_score_plan(const mfsdp_param_t* params, size_t n_params, int world_size, const int32_t* owner, size_t n_roles,
                     mfsdp_rank_score_t* rank_out, mfsdp_block_score_t* block_out, size_t block_cap, size_t* n_blocks);

/* Owner-segment gradient-reduction schedule ("each rank contributes its local full-gradient buffer, but
 * the reduced result is written only to the nonempty owner segment"; "deterministic native send/recv
 * schedules ... Cross-rank validation checks that every rank derives the same deterministic schedule and segment sizes
 * before communication begins").  The same records, in forward block order (reverse_blocks = 0), are the
 * materialisation schedule: the owner of a role sends its segment to the W - 1 ranks that need the full parameter.
 * HOST, integers.  DESIGN.md reading F1: one reduce-to-owner per role (on one NVSwitch
 * domain: ncclReduce with root = owner, or grouped send/recv), blocks in reverse model order when reverse_blocks != 0
 * (backward produces the last block first), roles of a block in parameter order.  Every rank calls this with the same
 * (params, world_size, owner) and compares *hash_out (FNV-1a 64 over the records) with its peers before it communicates;
 * a mismatch is a configuration error to raise, not a hang to wait for.
 *   owner_elem_off  where the reduced segment lands: element offset in the OWNER's rank-flat buffer of its kind (the
 *                   elem_off of that rank's descriptor table, mfsdp_plan);
 *   flag            position of the matrix among the owner's MATRIX descriptors = the index of its "gradient landed"
 *                   flag for mfsdp_muon_step_gated (-1 for tails).
 * ops_out == NULL: only *n_ops and *hash_out are written.  Errors as mfsdp_score_plan. */
typedef struct {
  uint32_t seq, role, kind, block_id, param_id, owner, dtype;
  int32_t  flag;
  uint64_t numel, owner_elem_off;
} mfsdp_reduce_op_t;
int mfsdp_reduce_schedule(const mfsdp_param_t* params, size_t n_params, int world_size, const int32_t* owner,
                          size_t n_roles, int reverse_blocks, mfsdp_reduce_op_t* ops_out, size_t ops_cap, size_t* n_ops,
                          uint64_t* hash_out);

/* Validate a descriptor table against PAPER.md:71 / Alg. 1 line 5 (HOST).  0 or MFSDP_ELAYOUT / MFSDP_EINVAL. */
int mfsdp_validate_desc(const mfsdp_desc_t* desc, size_t n_desc);

/* Elements spanned by the rank-flat matrix space and tail space of a descriptor table (HOST): what the caller
 * must allocate for W/G/M (matrix_elems) and P/G/m/v (tail_elems).  Either out pointer may be NULL. */
int mfsdp_flat_elems(const mfsdp_desc_t* desc, size_t n_desc, uint64_t* matrix_elems, uint64_t* tail_elems);

/* ---- Muon step (DEVICE work, HOST call) ----------------------------------------------------------------------- */
/* Bytes of DEVICE workspace mfsdp_muon_step needs for this table and precision (HOST). */
int mfsdp_workspace_bytes(const mfsdp_desc_t* desc, size_t n_desc, int precision, size_t* bytes);

/* Where the step leaves its per-matrix intermediates inside the workspace (HOST; for tests and callers that
 * consume the orthogonalised update): for the `index`-th MATRIX descriptor of the table,
 *   *o_byte_off   byte offset of O = X_K, stored rows x cols row-major exactly like the parameter (tall matrices
 *                 are NOT physically transposed: the kernels iterate X <- X (aI + bA' + cA'^2), A' = X^T X, which
 *                 is the transposed problem of the north_star read through the tensor-core operand descriptors),
 *                 row pitch *o_pitch elements of bf16 (MFSDP_NS_BF16) or float (MFSDP_NS_FP32);
 *   *ssq_byte_off byte offset of a double holding ||U||_F^2.
 * Any out pointer may be NULL. */
int mfsdp_workspace_view(const mfsdp_desc_t* desc, size_t n_desc, int precision, int ns_steps, size_t index,
                         size_t* o_byte_off, size_t* o_pitch, size_t* ssq_byte_off);

/* One owner-local Muon step on every MATRIX descriptor of the table (tail descriptors are ignored: routing,
 * PAPER.md:97).  For each matrix (SURVEY.md 8(c) O-2 / DESIGN.md section 2):
 *   M <- mu M + (1-mu) G ; U = (1-mu) G + mu M (Nesterov) or M ; X0 = U^(T if tall) / max(||U||_F, eps) ;
 *   K x { A = X X^T ; B = b A + c A A ; X <- a X + B X } ; O = X_K ; W <- W (1 - lr wd) - lr s(rows, cols) O.
 *   desc, n_desc   HOST in.    descriptor table (as returned by mfsdp_plan).  All matrix descriptors must share
 *                              one dtype.
 *   W              DEVICE i/o. rank-flat weights, dtype of the descriptors, 128-byte aligned base.
 *   G              DEVICE in.  rank-flat gradients, same dtype and offsets as W.
 *   M              DEVICE i/o. rank-flat momentum, always float, same element offsets.
 *   workspace      DEVICE.     >= mfsdp_workspace_bytes, 1024-byte aligned; contents need not be preserved
 *                              between calls; after the call it holds ||U||^2 and -- if hp->flags has
 *                              MFSDP_STEP_KEEP_O, or the update could not be fused -- O (mfsdp_workspace_view).
 *                              With bf16 weights and every cols % 8 == 0 (MFSDP_NS_BF16) the weight update runs
 *                              inside the last Newton-Schulz epilogue straight from the accumulator tile, and O is
 *                              written out only on request; the result is bit-identical to the separate passes.
 *                              May be NULL (and W, G, M too) when the table holds no matrix: the call is a no-op.
 *   cuda_stream    cudaStream_t (NULL = the legacy default stream).  Work is enqueued, not awaited.  After one
 *                              ordinary call with the same (table, workspace, precision) -- which builds the cached
 *                              launch tables with cudaMalloc / cudaMemcpy -- the step is CUDA-graph capturable (one
 *                              memset node and the kernel launches).  The hyper-parameters are baked into the
 *                              captured kernel arguments: re-capture when lr, momentum, ... change (for AdamW the
 *                              bias correction depends on hp->step, so every step needs its own capture or an
 *                              eager call).
 *                              The library caches, per (device, table contents, WORKSPACE POINTER, precision), a few
 *                              KB..MB of launch tables (TMA tensor maps hold the workspace address; tile lists) in
 *                              device memory of its own.  Entries are never evicted (launches in flight and captured
 *                              graphs reference them): keep the workspace pointer stable across steps.  After 1024
 *                              distinct keys the call fails with MFSDP_ECACHE until mfsdp_release_plans() is called.
 *   hp             HOST in.
 * Returns MFSDP_EINVAL (null / misaligned pointer, bad hyper-parameter, mixed dtypes), MFSDP_ECAP (ws_bytes too
 * small), MFSDP_ELAYOUT, MFSDP_EARCH (current device is not compute capability 10.x), MFSDP_ECUDA, MFSDP_ECACHE.
 * Thread safety: step functions may be called from several host threads (the cache is locked; counters are atomic;
 * mfsdp_strerror(MFSDP_ECUDA) is per calling thread).  mfsdp_tune, mfsdp_debug_trace and mfsdp_release_plans must not
 * run concurrently with step calls. */
int mfsdp_muon_step(const mfsdp_desc_t* desc, size_t n_desc, void* W, const void* G, void* M,
                    void* workspace, size_t ws_bytes, const mfsdp_muon_hparams_t* hp, void* cuda_stream);

/* mfsdp_muon_step whose momentum pass starts on each matrix as soon as that matrix' gradient has landed (PAPER.md:47,
 * 83: the gradient reduction "deposits the complete gradient on that owner"): the step may be
 * enqueued while the reduction is still running on another stream.
 *   ready   DEVICE in.  one uint32 per MATRIX descriptor, in table order.  The chunks of matrix i are processed once
 *                       ready[i] >= epoch (acquire at system scope, so that writes of a copy engine, a peer GPU or
 *                       the host made before the flag write are visible); G is read through L2 only.
 *   epoch               the value the producer writes for this step (e.g. the step number; flags never need a reset).
 * The matrices are taken in the order their flags go up, whatever the table order: each waiting thread block sweeps the
 * matrices it has chunks of and works on those that have landed (with the reverse-block order of mfsdp_reduce_schedule
 * the last matrices of the table land first).  The order changes no value.
 * The producer -- the reduction's completion, or a host-to-device copy -- raises flag i with
 * mfsdp_signal_ready(ready, i, epoch, producer_stream) AFTER the work that fills matrix i's gradient, on the stream
 * that does that work.  The producer's work must not depend on SM resources that the waiting kernel occupies: enqueue
 * the producer BEFORE this call (a kernel already running keeps its SMs), or use copy engines.  A wait longer than
 * ~10 s of SM clocks traps (MFSDP_ECUDA on the next call) instead of hanging the device.  The launch tables of a new
 * (table, workspace) are built -- synchronously -- before the first kernel of the call is enqueued, so the call never
 * blocks the host behind its own waiting kernel.  Newton-Schulz and the update
 * start when the whole momentum pass is done (stream order).  Results are bit-identical to mfsdp_muon_step. */
int mfsdp_muon_step_gated(const mfsdp_desc_t* desc, size_t n_desc, void* W, const void* G, void* M,
                          void* workspace, size_t ws_bytes, const mfsdp_muon_hparams_t* hp,
                          const uint32_t* ready, uint32_t epoch, void* cuda_stream);
/* Stream-ordered 32-bit write ready[index] = epoch (cuStreamWriteValue32: no kernel, no SM). */
int mfsdp_signal_ready(uint32_t* ready, size_t index, uint32_t epoch, void* cuda_stream);

/* mfsdp_muon_step that also writes every updated matrix into a second destination: the single-GPU half of the owner
 * fan-out ("ranks with nonempty segments send only those segments to the ranks that need the full parameter
 * for the current FSDP unit; in the common matrix case this is an owner fanout").  The weight-update
 * epilogue stores each 16-byte vector of the new W twice: into the owner's shard W and into fanout[i], the full-
 * parameter buffer of matrix i (rows x cols, row-major, 16-byte aligned, dtype of W).  The destination is an ordinary
 * device address as far as the kernels are concerned: a local buffer (what the tests use), peer memory mapped over
 * NVLink, or an NVSwitch multicast address, in which case the one store reaches every peer and no separate collective
 * follows the step.  (Mapping such memory is the caller's business; nothing here was measured on more than one GPU.)
 *   fanout   HOST in.  one DEVICE pointer per MATRIX descriptor, in table order; NULL entries = no copy for that matrix.
 * The transfer order for non-multicast fan-out is the forward-order schedule of mfsdp_reduce_schedule
 * (reverse_blocks = 0); its per-block cost estimate is C_B^owner of mfsdp_score_plan.  Not CUDA-graph capturable (the
 * destination table is copied from the host array on every call).  The device copy of that table belongs to the cached
 * launch tables of (table, workspace): fan-out calls that share them must be ordered on ONE stream -- a second call on
 * another stream or thread would overwrite the table under the first call's kernels (they share the workspace anyway).
 * Bit-identical W to mfsdp_muon_step. */
int mfsdp_muon_step_fanout(const mfsdp_desc_t* desc, size_t n_desc, void* W, const void* G, void* M,
                           void* workspace, size_t ws_bytes, const mfsdp_muon_hparams_t* hp,
                           void* const* fanout, void* cuda_stream);

/* Individual passes of the step, exposed so tests can check each kernel against the oracle and bench.py can time
 * them.  Same arguments and errors as mfsdp_muon_step.
 *   momentum pass: M, X~ = cast(U) in the workspace, ||U||^2.
 *   ns pass:       X_K from X~ and ||U||^2 (a2 + a3).
 *   update pass:   W from O (a4). */
int mfsdp_muon_momentum_pass(const mfsdp_desc_t* desc, size_t n_desc, const void* G, void* M,
                             void* workspace, size_t ws_bytes, const mfsdp_muon_hparams_t* hp, void* cuda_stream);
int mfsdp_muon_ns_pass(const mfsdp_desc_t* desc, size_t n_desc, void* workspace, size_t ws_bytes,
                       const mfsdp_muon_hparams_t* hp, void* cuda_stream);
int mfsdp_muon_update_pass(const mfsdp_desc_t* desc, size_t n_desc, void* W, void* workspace, size_t ws_bytes,
                           const mfsdp_muon_hparams_t* hp, void* cuda_stream);

/* The same step with HOST buffers (pinned for overlap; pageable works, serialised by the driver): copies G (and W, M
 * when `upload_state` == 1) to the caller's device staging buffers dW/dG/dM (128-byte aligned), runs the step on
 * `cuda_stream`, copies W and M back and synchronises the stream before returning.  upload_state: 1 = W and M travel
 * both ways every step; 0 = W and M stay in dW / dM between calls (only G goes up), both still come back; 2 = as 0 but
 * the momentum never leaves the device (hM may be NULL): G up, W down -- the traffic of a deployment that keeps the
 * optimizer state in HBM.  The resident set is cut into up
 * to 8 groups of consecutive matrices which are pipelined over two internal copy streams and the caller's stream: the
 * upload of group g + 1, the step of group g and the download of group g - 1 overlap (PCIe is full duplex; inside a
 * group W rides in under Newton-Schulz and M goes out right after the momentum pass).  That needs one workspace slice
 * per group: pass a workspace of mfsdp_host_workspace_bytes (a few KB more than mfsdp_workspace_bytes); with a smaller
 * one the call still works, as a single group.  Everything is ordered after the work already queued on
 * `cuda_stream`.  Results are bit-identical to mfsdp_muon_step.  Used for the end-to-end measurement. */
int mfsdp_host_workspace_bytes(const mfsdp_desc_t* desc, size_t n_desc, int precision, size_t* bytes);
int mfsdp_muon_step_host(const mfsdp_desc_t* desc, size_t n_desc, void* hW, const void* hG, void* hM,
                         void* dW, void* dG, void* dM, int upload_state,
                         void* workspace, size_t ws_bytes, const mfsdp_muon_hparams_t* hp, void* cuda_stream);

/* ---- momentum pass of one matrix for callers that may not allocate (DEVICE work, HOST call) ----------------------
 * Every step call above builds device-side launch tables with cudaMalloc the first time it sees a (table, workspace)
 * pair and needs a caller-allocated workspace.  Some callers of an owner-local optimizer can do neither: a trainer
 * whose framework allocator has already claimed the GPU up to its planned budget (a raw cudaMalloc may fail or break a
 * memory limit the job runs under); code inside the step loop while the gradient reduction of PAPER.md:83 is still in
 * flight on another stream (cudaMalloc / cudaFree synchronise the whole device and would stall that overlap); a hook
 * of a host library that forbids CUDA memory management.  For them this call runs SURVEY.md 8(a) a1 and the scalar
 * part of a2 on ONE matrix with no allocation, no host-to-device copy and no cached table:
 *   M <- mu M + (1-mu) G ; U = (1-mu) G + mu M (hp->nesterov != 0) or M ; X = cast(U) ;
 *   *ssq = ||U||_F^2 ; *inv_norm = 1 / max(||U||_F, hp->eps).
 * The one piece of scratch the pass needs (a double per 16384-element chunk, between the streaming kernel and the
 * fixed-order reduction) lives in a fixed array inside the library's device image.
 *   rows, cols   the matrix, row-major and contiguous (G, M and X all have row pitch = cols); rows * cols must not
 *                exceed mfsdp_static_max_elems() = 2^30, else MFSDP_ETOOBIG is returned and nothing is launched.
 *   dtype        MFSDP_BF16 | MFSDP_F32: element type of G.
 *   precision    MFSDP_NS_BF16 -> X is bf16, MFSDP_NS_FP32 -> X is float.
 *   G            DEVICE in.   rows * cols elements, 16-byte aligned.
 *   M            DEVICE i/o.  rows * cols floats, 16-byte aligned, updated in place.
 *   X            DEVICE out.  rows * cols elements of bf16 / float, 16-byte aligned.
 *   ssq          DEVICE out.  one double (8-byte aligned).
 *   inv_norm     DEVICE out.  one float.
 *   hp           HOST in.     only momentum, nesterov and eps are read.
 * What to know before relying on it:
 *   - the array is 512 KiB and every GPU that loads libmfsdp holds it until the process exits, used or not;
 *   - the FIRST call on each device does the set-up (looks up the array's device address with that device current and
 *     makes the runtime load the library's device code); make that call before any stream capture starts.  Later
 *     calls only enqueue two kernels on cuda_stream and return without synchronising;
 *   - all calls on a device share the array, and it keeps the previous call's contents.  Nothing in it has to start at
 *     zero (each call writes every partial it reads), so calls ordered on one stream, or by events, are safe back to
 *     back; two calls that may run at the same time on one GPU overwrite each other's partials and race;
 *   - M, X and ||U||^2 are bit-identical to mfsdp_muon_momentum_pass on a table holding the same matrix.
 * Returns MFSDP_EINVAL (null / misaligned pointer, zero dimension, bad dtype / precision / momentum / eps),
 * MFSDP_ETOOBIG, MFSDP_EARCH, MFSDP_ECUDA. */
uint64_t mfsdp_static_max_elems(void);
int mfsdp_momentum_pass_static(uint32_t rows, uint32_t cols, int dtype, int precision, const void* G, void* M, void* X,
                               double* ssq, float* inv_norm, const mfsdp_muon_hparams_t* hp, void* cuda_stream);

/* ---- AdamW on packed tails (DEVICE work, HOST call) ------------------------------------------------------------
 * For every TAIL descriptor (matrix descriptors are ignored), element-wise:
 *   p <- p (1 - lr wd) ; m <- b1 m + (1-b1) g ; v <- b2 v + (1-b2) g^2 ;
 *   p <- p - lr (m / (1 - b1^t)) / (sqrt(v / (1 - b2^t)) + eps).
 *   P, G   DEVICE. rank-flat tail parameters / gradients, dtype of the descriptors (one dtype for all tails).
 *   m, v   DEVICE. rank-flat first / second moments, always float, same element offsets.
 * Returns as mfsdp_muon_step (hp->step < 1 is MFSDP_EINVAL). */
int mfsdp_adamw_tail_step(const mfsdp_desc_t* desc, size_t n_desc, void* P, const void* G, void* m, void* v,
                          const mfsdp_adamw_hparams_t* hp, void* cuda_stream);

/* ---- owner-local Shampoo on the same descriptors (DEVICE work, HOST call) ---------------------------------------
 * "The owner-placement runtime is optimizer-agnostic: each 2D matrix is whole on its owner, so any
 * single-device matrix optimizer runs there with no gather and no distributed variant.  We verify this by swapping
 * owner-Muon for Shampoo (full L/R preconditioners with inverse fourth root) ... float32".  The
 * paper prints neither formulas nor hyper-parameters; what is computed is Algorithm 1 of Gupta et al. (2018) for
 * matrices under the readings S1-S7 of DESIGN.md section 4.  For every MATRIX descriptor (tails are ignored):
 *   S1  L <- beta2 L + w G G^T ;  R <- beta2 R + w G^T G ;  w = 1 if beta2 == 1 (running sum) else 1 - beta2
 *   S2  ridge relative to the mean eigenvalue: S~ = S + rho I, rho = eps tr S / d ;  tr S <= 0 -> the preconditioner is I
 *   S7  float32 floor of the ridge: rho = max(eps tr S / d, eps_floor ||S||_F).  The statistic carries rounding noise of
 *       about 2^-22 ||S||_F in this arithmetic; a ridge below it leaves S~ indefinite (rank-deficient statistics: every
 *       wide or tall matrix) and no float32 iteration can then return S~^{-1/4}.  eps_floor = 2^-20 keeps the condition
 *       number below 2^20; 0 = the plain S2 (a root that meets a NaN falls back to (tr S / d + rho)^{-1/4} I, flagged)
 *   S3  P_L = L~^{-1/4}, P_R = R~^{-1/4}
 *   S4  D = P_L G P_R ;  W <- W (1 - lr weight_decay) - lr D
 *   S5  the roots are recomputed at steps with (step - 1) % root_every == 0, from statistics that include G_step;
 *       other steps reuse the stored roots
 *   S6  the roots are computed by the coupled Newton iteration  M_0 = z S~, X_0 = z^{1/4} I, z = 5 / (2 bound),
 *       bound = min(||S||_F, 1.6 |S x_8|) + rho (x_8: eight power-iteration steps from a fixed start vector),
 *       T = (5 I - M) / 4, X <- X T, M <- T^4 M.  The first iterations additionally scale M by 2.5 and X by 2.5^(1/4):
 *       every eigenvalue of M is <= 1 after an iteration, so the scaled M stays inside the convergence region and its
 *       small eigenvalues grow 6.1 x instead of 2.44 x per iteration.  It stops at max |M - I| < root_tol, when the error
 *       no longer falls (fp32-class noise floor) or after max_root_iters; X -> S~^{-1/4}.  11-13 iterations.
 * Arithmetic: every matrix product runs on the bf16 tensor cores with fp32 values carried as three bf16 terms
 * (24 significand bits, fp32 exponent range) and fp32 accumulation -- fp32-class, not bit-identical to an fp32 FFMA loop;
 * the two products of S4 carry their operands to two terms (2^-16-class: the roots are no more accurate than 1e-3).
 * L and R are fp32; P_L, P_R are kept as three bf16 planes (their sum is the fp32 value).  Dynamic range: G G^T is
 * accumulated in fp32, so rms(G) must stay within about 1e-17 .. 1e+16 (as for the Muon path); inside it the first step's
 * D is invariant under power-of-two scalings of G bit for bit (tested).
 *   W, G        DEVICE.  rank-flat matrix parameters (in/out) / gradients (in), 16-byte aligned; dtype of the descriptors.
 *   state       DEVICE in/out.  mfsdp_shampoo_state_bytes, 1024-byte aligned, caller-owned, ZEROED before the first
 *                               step (L_0 = R_0 = 0); layout per matrix: mfsdp_shampoo_view.
 *   workspace   DEVICE scratch. 1024-byte aligned; at least min_bytes of mfsdp_shampoo_workspace_bytes.  The roots of the
 *                               resident set are computed in groups of as many (L, R) problems as fit behind the fixed part:
 *                               full_bytes processes them all at once (fewest launches), min_bytes one at a time.
 *   hp          HOST in.
 * Enqueues on cuda_stream and does not synchronise (the number of launches is fixed: converged problems are skipped
 * on the device).  Launch tables are cached per (table, state, workspace, ws_bytes, flags); at most 64 keys
 * (MFSDP_ECACHE beyond; mfsdp_release_plans frees them).  W and G may be other buffers from call to call: the records that
 * hold their addresses are re-pointed and re-uploaded in stream order (a few hundred KB, only when they change; calls
 * on one table must then be ordered on one stream).  A captured CUDA graph keeps the addresses it was captured with.
 * Errors as mfsdp_muon_step. */
enum { MFSDP_SHAMPOO_KEEP_D = 1u };      /* flags bit0: also leave D = P_L G P_R (fp32) in the workspace              */
typedef struct {
  double  lr;              /* eta                                                                                  */
  double  weight_decay;    /* lambda (decoupled)                                                                   */
  double  beta2;           /* in (0, 1]; 1 = running sum (Gupta et al.), < 1 = moving average (Anil et al.)        */
  double  eps;             /* relative ridge, >= 0 (1e-6)                                                          */
  double  eps_floor;       /* S7, >= 0 (2^-20)                                                                     */
  double  root_tol;        /* 0 -> 1e-6                                                                            */
  int64_t step;            /* 1-based                                                                              */
  int32_t root_every;      /* >= 1                                                                                 */
  int32_t max_root_iters;  /* 0 -> ceil(log(0.08 / eps_floor) / log(6.1)) + 9 (16 at 2^-20), 40 without a floor     */
  uint32_t flags;          /* MFSDP_SHAMPOO_*                                                                      */
  uint32_t reserved;       /* 0                                                                                    */
} mfsdp_shampoo_hparams_t;
int mfsdp_shampoo_state_bytes(const mfsdp_desc_t* desc, size_t n_desc, size_t* bytes);
int mfsdp_shampoo_workspace_bytes(const mfsdp_desc_t* desc, size_t n_desc, uint32_t flags, size_t* min_bytes,
                                  size_t* full_bytes);
int mfsdp_shampoo_step(const mfsdp_desc_t* desc, size_t n_desc, void* W, const void* G, void* state, size_t state_bytes,
                       void* workspace, size_t ws_bytes, const mfsdp_shampoo_hparams_t* hp, void* cuda_stream);
/* Layout of the `index`-th matrix (HOST; tests and callers that checkpoint the state):
 * out[0..3] = byte offsets in `state` of L (rows x out[4] floats), R (cols x out[5] floats), P_L (3 planes of
 * rows x out[4] bf16, out[6] elements apart), P_R (3 planes of cols x out[5] bf16, out[7] elements apart);
 * out[8] = byte offset in the workspace of D (rows x out[5] floats; MFSDP_SHAMPOO_KEEP_D only);
 * out[9] = byte offset in the workspace of the root control records of this matrix (L then R), out[10] bytes each:
 *   { double tr, fro2; float rho, z, x0, last_err; uint32 err_bits, iters, done, identity;
 *     float alpha_m, alpha_x; uint32 n_scaled, pad }  with done = 1 converged (max |M - I| < root_tol, or at the fp32-class
 *     noise floor), 2 the iteration met a NaN (S~ not positive definite in this arithmetic: the root was REPLACED by the
 *     scalar (tr S / d + rho)^{-1/4} I), 3 max_root_iters reached first (P is the last iterate, not a converged root);
 * out[11] = byte offset in the workspace of the status record of the last step that recomputed roots:
 *   uint32 { converged, not_positive_definite, out_of_budget, roots } over the whole resident set.  mfsdp_shampoo_step
 *   itself returns MFSDP_OK in all three cases (it never synchronises): a caller that must know whether the method's
 *   own roots were used reads these 16 bytes after the step -- anything but {roots, 0, 0, roots} means some
 *   preconditioner is a substitute. */
int mfsdp_shampoo_view(const mfsdp_desc_t* desc, size_t n_desc, uint32_t flags, size_t index, size_t out[12]);

/* Debug / test aid (HOST): byte offsets inside the workspace of the `index`-th matrix' NS buffers:
 * out[0], out[1] = X ping-pong buffers (X~ = cast(U) is written to out[0]; rows x cols like the parameter),
 * out[2] = A (d x d, d = min(rows, cols)), out[3] = P = aI + bA + cA^2 (d x d),
 * out[4] = X row pitch in elements, out[5] = A/P row pitch in elements. */
int mfsdp_debug_ws_offsets(const mfsdp_desc_t* desc, size_t n_desc, int precision, size_t index, size_t out[6]);

/* Frees every cached launch table of the process after synchronising their devices (HOST).  The caller guarantees
 * that no CUDA graph captured from a step call will be replayed afterwards.  Always MFSDP_OK. */
int mfsdp_release_plans(void);

/* Which Newton-Schulz kernel class a rows x cols matrix runs in under MFSDP_NS_BF16 with the current knob values (HOST):
 * 0 = a whole-matrix kernel (A and P stay on chip: the A / P workspace buffers of mfsdp_debug_ws_offsets are NOT written),
 * 1 = single-CTA tiles, 2 = CTA-pair tiles.  Negative code on rows == 0 or cols == 0. */
int mfsdp_ns_class(uint32_t rows, uint32_t cols);

/* ---- tuning knobs (HOST) -------------------------------------------------------------------------------------
 * Scheduling choices of the tensor-core Newton-Schulz path.  They change HOW tiles are formed and ordered, never
 * what is computed (tests run the parity suite under several settings).  Setting a knob synchronises the device
 * and drops the cached launch tables, which are rebuilt on the next step.  The values below are the only initial
 * state (no environment variables).
 *   MFSDP_TUNE_PAIR_MIN_D   matrices with min(rows, cols) >= value run on CTA pairs (tcgen05 cta_group::2,
 *                           256 x 512 output tiles held as two 256-column TMEM accumulators, 256 x 256 in phases
 *                           with a short k loop); smaller ones on single CTAs (128 x N tiles).  default 1024
 *                           (measured: GPT-2 768-row matrices run 14 % faster on single CTAs, 1024-row Llama k / v
 *                           projections equally fast either way)
 *   MFSDP_TUNE_SYM_BAND     row blocks per band of the symmetric (GRAM, POLY) tile order, single-CTA class.  16
 *   MFSDP_TUNE_SYM_BAND2    the same for the CTA-pair class.  8
 *   MFSDP_TUNE_RECT_GROUP   column tiles per panel of the rectangular (APPLY) tile order.  4
 *   MFSDP_TUNE_WIDE_MIN_KB  CTA-pair tiles are 512 columns wide (else 256) in phases whose k loop has at least this
 *                           many 64-element blocks.  8
 *   MFSDP_TUNE_FUSED_BELOW_D matrices with min(rows, cols) < value whose padded X fits 128 KB of shared memory run in
 *                           the whole-matrix kernel (one CTA keeps X, A and P on chip for all K iterations); 1 switches
 *                           that kernel off.  129
 *   MFSDP_TUNE_FUSED2_BELOW_D matrices with 128 < min(rows, cols) < value (<= 257) and max(rows, cols) <= 512 run in
 *                           the second whole-matrix kernel (one CTA keeps A and P on chip for all K iterations and
 *                           streams X through shared memory); 1 switches that kernel off.  257
 * Returns MFSDP_EINVAL for an unknown knob or value < 1; mfsdp_get_tune returns the value or a negative code. */
enum { MFSDP_TUNE_PAIR_MIN_D = 0, MFSDP_TUNE_SYM_BAND = 1, MFSDP_TUNE_SYM_BAND2 = 2, MFSDP_TUNE_RECT_GROUP = 3,
       MFSDP_TUNE_WIDE_MIN_KB = 4, MFSDP_TUNE_FUSED_BELOW_D = 5, MFSDP_TUNE_FUSED2_BELOW_D = 6, MFSDP_TUNE_COUNT_ = 7 };
int mfsdp_tune(int knob, int value);
int mfsdp_get_tune(int knob);

/* Debug aid: tile trace of the tensor-core Newton-Schulz kernels.  dev_buf: DEVICE buffer of `bytes` bytes, 8-byte
 * aligned, zeroed by the caller and owned by the caller; NULL switches tracing off (the default).  While set, every
 * NS tile appends one record of six 64-bit words after the counter word dev_buf[0]:
 *   (phase index 3 * iteration + {0 GRAM, 1 POLY, 2 APPLY} << 32 | tile index within the launch), (walking unit << 32 | SM id),
 *   %globaltimer ns when the tile's accumulator was complete, %globaltimer ns when its first epilogue warp was done,
 *   the SM's clock64 at the first instant, (k blocks of the tile << 32 | UMMA N).
 * The CTA-pair GEMM of the Shampoo step (k_sgemm3p) appends, per tile and per role of the pair's leader CTA, a record
 *   (role {0 TMA producer, 1 UMMA issuer, 2 first epilogue warp} << 32 | tile index), clock64 at the start and at the
 *   end of the role's work on the tile, cycles spent waiting (producer: for a free ring stage; issuer: for a folded
 *   TMEM accumulator; epilogue: for a complete accumulator), a second figure (issuer: cycles waiting for operands;
 *   epilogue: cycles until its stores began), SM id.
 * Records beyond the capacity are dropped (the counter keeps counting).  Returns MFSDP_EINVAL on a misaligned or
 * too-small buffer. */
int mfsdp_debug_trace(void* dev_buf, size_t bytes);

/* ---- misc ----------------------------------------------------------------------------------------------------- */
const char* mfsdp_strerror(int code);      /* static string; for MFSDP_ECUDA the calling thread's last CUDA error */
int mfsdp_version(void);                   /* ABI version, currently 2                                            */
/* Number of kernels the library launched since process start (for bench.py's gpu_launches claim). */
uint64_t mfsdp_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* MFSDP_H_ */

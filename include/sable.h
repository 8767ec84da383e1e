/*
 * sable.h -- C ABI of the B200-native batched Newton-Raphson AC power-flow library
 * (hot path of SABLE, arxiv/paper_2606_07099; PAPER.md = text of the paper).
 *
 * What the library computes (per scenario b of a batch sharing one network):
 *   Step-1 equations  F1(z1) = [P_i(V) - P_spec,i  (i not slack);  Q_i(V) - Q_spec,i  (i PQ)] = 0     (eq. 6)
 *   with S = V o conj(Y_bus V), V_i = Vm_i e^{j theta_i}, unknowns z1 = [theta (non-slack); Vm (PQ)]  (eq. 4)
 *   Newton step       J1(z1_t) dz = -F1(z1_t),  z1_{t+1} = z1_t + dz                                  (eq. 7-8)
 *   adjoint           J1(z1*)^T lambda = g                                                            (eq. 14)
 * Sign convention: F = S_calc - S_spec (BASELINE.json north_star); the paper writes spec - calc
 * (PAPER.md:55): the Newton step is identical, lambda here = -lambda_paper = d(g^T z1)/dS_spec.
 *
 * Units: per-unit and radians.  One slack bus.  No Q-limits, taps or shunts beyond what Y_bus carries.
 * Threading: a context may be used by one host thread at a time.  Errors never abort or throw;
 * every call returns a sable_status and leaves a message retrievable with sable_last_error().
 */
#ifndef SABLE_H
#define SABLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sable_ctx sable_ctx;          /* opaque; owned by the library */

typedef enum {
    SABLE_OK = 0,
    SABLE_ERR_INVALID_ARG = 1,               /* null pointer, negative size, batch > max_batch, bad option */
    SABLE_ERR_STRUCTURE = 2,                 /* malformed CSR, bus_type/slack inconsistent, bus not connected to the slack */
    SABLE_ERR_ALLOC = 3,                     /* host or device allocation failed */
    SABLE_ERR_CUDA = 4,                      /* CUDA runtime error (launch, copy, no device) */
    SABLE_ERR_STATE = 5                      /* e.g. sable_adjoint before a sable_solve that kept factors */
} sable_status;

enum { SABLE_BUS_PQ = 0, SABLE_BUS_PV = 1, SABLE_BUS_SLACK = 2 };
enum { SABLE_FP64 = 0, SABLE_MIXED = 1 };    /* MIXED: FP64 mismatch / state, FP32 Jacobian factors and solves (Table I) */
enum { SABLE_MODE_FUSED = 0, SABLE_MODE_STAGED = 1 };

/* Launch tuning.  Every field has an "automatic" value (what sable_default_options() returns); the library then chooses
 * from the grid size, the level structure and max_batch.  For experiments each field can also be
 * overridden through the environment variable named beside it (read at sable_create, only when the field is left automatic;
 * values are clamped to the stated range). */
typedef struct {
    int32_t group;            /* scenarios a CTA advances in lockstep = group size of the interleaved workspace: 1, 2, 4 ... 32;
                                 0 = automatic                                                        (SABLE_G) */
    int32_t ctas_per_sm;      /* cap on resident CTAs per SM of the NR kernel, 1 ... 32; 0 = automatic  (SABLE_CTAS) */
    int32_t on_chip;          /* 1 = all arrays of every slot in shared memory (if they fit), 0 = HBM workspace,
                                 -1 = automatic                                                       (SABLE_ONCHIP) */
    int32_t ring_slots;       /* on-chip placement: slots of the level-blob ring, 0 ... 8 (0 = off); -1 = automatic  (SABLE_RING_R) */
    int32_t ring_slot_bytes;  /* bytes per ring slot, 256 ... 65536; -1 = automatic                     (SABLE_RING_SLOT) */
    int32_t front_nodes;      /* HBM placement: cap on the nodes of the dense top front, 0 ... 96 (0 = off); -1 = automatic  (SABLE_FRONT) */
    int32_t front_kb;         /* shared-memory budget of the front per CTA in KB, 0 ... 220; -1 = automatic  (SABLE_FRONT_KB) */
    int32_t threads_stage;    /* threads per CTA of the staged kernels, 32 ... 1024; 0 = automatic       (SABLE_THREADS1) */
    int32_t threads_lin;      /* threads per CTA of the adjoint kernel, 32 ... 1024; 0 = automatic      (SABLE_THREADS_LIN) */
    int32_t timing;           /* 1 = per-phase cycle counters of CTA 0 (sable_debug_timing)            (SABLE_TIMING) */
    int32_t cluster;          /* HBM placement: CTAs (one thread-block cluster) that serve one group of scenarios together,
                                 1, 2, 4, 8; 0 = automatic (teams when the batch is too small to fill the SMs)  (SABLE_CLUSTER) */
} sable_tuning;

typedef struct {
    int32_t max_batch;      /* scenarios per sable_solve call; all device buffers are sized for it at create time, and the launch
                               plan (scenarios interleaved per CTA, threads) is made for a batch of THIS size: a context planned for a
                               large batch serves a much smaller one at about the large batch's latency -- create one context per
                               batch size in use, or fix the layout through tune.group / threads */
    int32_t precision;      /* SABLE_FP64 or SABLE_MIXED */
    int32_t keep_factors;   /* 1: after the NR loop, J1 is re-factored at the final iterate and the factors are kept
                               for sable_adjoint (reading 16) */
    int32_t mode;           /* SABLE_MODE_FUSED: one persistent kernel runs the whole NR loops of the batch;
                               SABLE_MODE_STAGED: one kernel per stage (mismatch + fill / refactor + solve), state in HBM
                               between stages, host check of the active count -- used for per-stage profiling */
    int32_t device;         /* CUDA device ordinal; -1 = host-only context (symbolic phase only: sable_get_info and the
                               sable_debug_* pattern queries work, solve / adjoint return SABLE_ERR_STATE) */
    int32_t threads;        /* threads per CTA for the NR kernel; 0 = library default for the grid size  (SABLE_THREADS) */
    int32_t ir_sweeps;      /* inner iterative-refinement sweeps of the forward linear solve, 0 ... 8 (default 0).  The paper's scheme
                               has none (Table I): the Newton loop with its FP64 residual and FP64 state
                               accumulation is the refinement (reading 15).  k > 0 (needs precision = SABLE_MIXED and
                               mode = SABLE_MODE_STAGED, else sable_create returns INVALID_ARG): after the FP32 solve of
                               J1 dz = -F1, k times r = -F1 - J1 dz with F1 and J1 evaluated in FP64 from Y_bus and the state
                               (nothing stored), J1 c = r on the same FP32 factors, dz += c in FP64; the step
                               then has FP64 accuracy and the iteration counts are those of an FP64 Newton loop.  Costs
                               2 + 3 k extra launches per iteration and nine [max_batch][n_bus] FP64 arrays (allocated at create).
                               FP64 refinement of the ADJOINT solve on FP32 factors: sable_adjoint_refined. */
    sable_tuning tune;
} sable_options;

/* Options with every field at its default / automatic value: max_batch 1, FP64, keep_factors 1, fused, device 0. */
sable_options sable_default_options(void);

typedef struct {
    int32_t n_bus, n_pq, n_pv;
    int32_t n;              /* scalar unknowns n_pv + 2 n_pq */
    int32_t nnz_y;          /* stored Y_bus entries after canonicalisation */
    int32_t nnz_j;          /* scalar nonzeros of J1 */
    int32_t nnz_lu;         /* scalar nonzeros of L+U on the static fill pattern (unit diagonal of L not counted) */
    int32_t n_node;         /* bus-level nodes = n_bus - 1 */
    int32_t n_pair;         /* bus-level off-diagonal block pairs {U(m,j), L(j,m)} in the filled pattern */
    int32_t n_pair_j;       /* of which structurally present in J1 (the rest is fill) */
    int32_t n_level;        /* elimination levels */
    int64_t n_term;         /* block multiply-subtract terms per refactorisation (pair targets) */
    int64_t n_term_diag;    /* ... (diagonal targets) */
    int64_t lu_flops;       /* scalar FP multiply-adds x2 per refactorisation on the unpadded pattern */
    int64_t factor_bytes;   /* bytes of one scenario's stored factors (padded 2x2 blocks, in factor precision) */
    int64_t bytes_iter_m0;  /* SURVEY.md §8(d) model M0: algorithmic HBM bytes per scenario per NR iteration */
    int64_t bytes_adjoint_m0; /* same for one adjoint solve */
    int32_t smem_bytes;     /* dynamic shared memory per CTA of the NR kernel */
    int32_t placement;      /* 0: factors, V and rhs of every slot in shared memory; 2: everything in the group-interleaved
                               HBM workspace */
    int32_t threads;        /* threads per CTA */
    int32_t ctas_per_sm;    /* occupancy the NR kernel was sized for */
    int32_t slots_per_cta;  /* scenarios a CTA of the NR kernel advances in lockstep */
    int32_t cut_level;      /* first elimination level kept in shared memory: 0 (placement 0) or n_level (placement 2) */
    int32_t front_k;        /* placement 2: nodes of the dense top front (the last elimination levels, factored as one dense
                               block matrix in shared memory); 0 = none */
    int32_t front_level;    /* first elimination level of that front (n_level if none) */
    int32_t threads_lin;    /* threads per CTA of the adjoint kernel */
    int32_t threads_stage;  /* threads per CTA of the staged kernels */
    int32_t cluster;        /* CTAs per team (thread-block cluster) of the NR kernel; 1 = every CTA works alone */
} sable_info;

/* Build the shared fixed-pattern template for one network (host symbolic phase, run once; PAPER.md:185-197:
 * "symbolic setup only once for a shared topology"): canonical Y_bus CSR, PV/PQ/slack index maps, minimum-degree
 * ordering of the bus graph, static block L+U fill pattern, elimination levels, multiply-subtract term lists and
 * Jacobian fill metadata; uploads it and allocates every device buffer for opt->max_batch scenarios.
 *   n_bus            number of buses (>= 2)
 *   row_ptr[n_bus+1], col_idx[nnz], y_re[nnz], y_im[nnz]   HOST.  Y_bus = G + jB in CSR; columns may be unsorted,
 *                    duplicates are summed, a missing diagonal or transpose entry is added with value 0.
 *   bus_type[n_bus]  HOST.  SABLE_BUS_PQ / PV / SLACK; exactly one slack, and it must equal `slack`.
 *   opt              may be NULL (= sable_default_options()).  Start from sable_default_options() and change fields:
 *                    a zero-initialised struct is NOT the default (on_chip / ring / front fields use -1 for automatic).
 *   out              receives the context.  The input arrays are not referenced after the call returns.
 * Errors: INVALID_ARG, STRUCTURE, ALLOC, CUDA.  On error *out = NULL (message via sable_last_error(NULL)). */
sable_status sable_create(int32_t n_bus, const int32_t* row_ptr, const int32_t* col_idx,
                          const double* y_re, const double* y_im, const uint8_t* bus_type, int32_t slack,
                          const sable_options* opt, sable_ctx** out);

/* Batched Newton-Raphson (eq. 6-8; loop convention DESIGN.md):
 *   it = 0; loop { r = ||F1(V)||_inf; if r <= tol: converged; if it == max_it or r not finite: stop; solve; update; ++it }
 * All arrays are DEVICE pointers, row-major [batch][n_bus], owned by the caller, not kept after the call.
 *   p_spec, q_spec   net injections P_spec = p_g - p_d, Q_spec = q_g - q_d.  p_spec is ignored at the
 *                    slack, q_spec is used at PQ buses only.
 *   v_set            |V| at PV and slack buses (the decision block x of eq. 3); ignored at PQ buses.
 *   vm0, va0         initial |V| (PQ buses) and angle (non-slack), or both NULL for the flat start (PAPER.md:287:
 *                    Vm = 1, theta = 0; PV/slack magnitudes at their setpoints, slack angle 0).
 *   vm, va           out: final |V| and angle (rad).  May not alias the inputs.
 *   iterations       out [batch] int32: Newton updates applied if converged, max_it otherwise.
 *   converged        out [batch] uint8.  Non-convergence is not an error.
 *   final_norm       out [batch] double or NULL: ||F1||_inf at the returned V.
 *   cuda_stream      cudaStream_t; the call only enqueues work (no host synchronisation in fused mode).
 * Converged scenarios stop consuming bandwidth (per-scenario masking).  Errors: INVALID_ARG, STATE, CUDA. */
sable_status sable_solve(sable_ctx* ctx, int32_t batch, const double* p_spec, const double* q_spec,
                         const double* v_set, const double* vm0, const double* va0, double tol, int32_t max_it,
                         double* vm, double* va, int32_t* iterations, uint8_t* converged, double* final_norm,
                         void* cuda_stream);

/* Adjoint J1^T lambda = g (eq. 14) on the factors kept by the last sable_solve (keep_factors = 1),
 * i.e. J1 at that call's final iterates; only transposed triangular solves run.
 *   g_va [batch][n_bus]  dl/dtheta_i (slack entry ignored);   g_vm [batch][n_bus]  dl/dVm_i (PQ entries used)
 *   lam_p, lam_q [batch][n_bus]  out: multipliers of the P_i / Q_i equations; 0 at the slack / off PQ buses.
 * A scenario whose kept factors carry a tiny-pivot flag (sable_get_pivot_flags, bit 1) gets NaN in every entry: static
 * pivoting failed there and, unlike the forward path, nothing downstream would reveal a wrong lambda.
 * All DEVICE pointers.  batch must equal the batch of the last solve.  Errors: INVALID_ARG, STATE, CUDA. */
sable_status sable_adjoint(sable_ctx* ctx, int32_t batch, const double* g_va, const double* g_vm,
                           double* lam_p, double* lam_q, void* cuda_stream);

/* Tiny-pivot flags of the last sable_solve (the paper's cuDSS path pivots internally; this library uses static
 * 2x2 block-diagonal pivots in a fixed order, shared by the batch): flags[b] bit 0 = in some refactorisation of scenario b a
 * pivot block D had |det D| <= eps * max|D_ij|^2 (eps = 1e-10 in FP64, 1e-6 with FP32 factors) or a non-finite
 * determinant; bit 1 = that happened in the LAST refactorisation (with keep_factors: in the kept factors).  A flagged
 * scenario that still converged is fine (the FP64 residual test protects the forward path); a flagged scenario that did not
 * converge should be re-solved by a pivoting solver.  flags [batch] int32 DEVICE out; asynchronous on the stream.
 * Errors: INVALID_ARG (batch differs from the last solve), STATE, CUDA. */
sable_status sable_get_pivot_flags(sable_ctx* ctx, int32_t batch, int32_t* flags, void* cuda_stream);

/* Step-2 explicit recovery (PAPER.md:80 eq. 5, :95-99 eq. 9: with dF2/dz2 = I the block z2 = [p_g at the slack; q_g at
 * PV and slack buses] is read off the mismatch rows that Step 1 does not use).  Returns the calculated net injections
 * P_i(V), Q_i(V) of S = V o conj(Y_bus V) for EVERY bus at the given voltages (normally the vm, va of sable_solve):
 * p_inj at the slack is the recovered slack injection, q_inj at PV / slack buses the recovered reactive injections
 * (generation = injection + load); at the other rows they equal the specified values up to the final
 * mismatch.  All DEVICE pointers, [batch][n_bus]; asynchronous on the stream; allocates nothing.  Grids above
 * 4 096 buses with batch x n_bus >= 2^18, and all grids above 10 240 buses, keep V in the context's workspace (that overwrites
 * the iterate of the last solve there, not the kept factors and not the caller's arrays).
 * Errors: INVALID_ARG, STATE, CUDA. */
sable_status sable_recover(sable_ctx* ctx, int32_t batch, const double* vm, const double* va, double* p_inj,
                           double* q_inj, void* cuda_stream);

/* Implicit-layer backward (eqs. 10-16): total derivative dL/dx of a scalar loss w.r.t. the layer input
 * x = [p_g at PV buses; Vm at PV and slack buses] (eq. 3), given the partials of L w.r.t. the completed buffer
 * y = [p_g, q_g at PV and slack buses; Vm; theta] (eq. 1) at the solution of the last sable_solve (keep_factors = 1):
 * one transposed SpMV with J2 (eq. 12), the adjoint solve of eq. 14 on the kept factors, one transposed SpMV with J3 and
 * the selector term (eq. 16).  With this library's sign F = S_calc - S_spec:  dL/dp_g,k = dL/dp_g,k|direct + lambda_P,k.
 *   vm, va                the vm, va returned by that sable_solve
 *   gl_pg, gl_qg          dL/dp_g,i and dL/dq_g,i: read at PV and slack buses (gl_pg at a PV bus is the direct partial
 *                         w.r.t. the input itself; at the slack it multiplies the recovered slack injection)
 *   gl_vm, gl_va          dL/dVm_i (all buses), dL/dtheta_i (slack entry ignored)
 *   dx_pg, dx_vm          out: dL/dp_g (nonzero at PV buses), dL/dVm (nonzero at PV and slack buses)
 * All DEVICE pointers, [batch][n_bus]; batch must equal the batch of the last solve; asynchronous on the stream; for
 * grids above 3 413 buses the state part of the workspace is used as scratch (the kept factors stay intact).
 * Errors: INVALID_ARG, STATE, CUDA. */
sable_status sable_layer_backward(sable_ctx* ctx, int32_t batch, const double* vm, const double* va,
                                  const double* gl_pg, const double* gl_qg, const double* gl_vm, const double* gl_va,
                                  double* dx_pg, double* dx_vm, void* cuda_stream);

/* Adjoint of eq. 14 with FP64 iterative refinement on the kept factors (Table I runs the backward LU in single
 * precision; this call brings lambda back to FP64 accuracy without an FP64 factorisation):
 *   lambda_0 = solve(g);  repeat `sweeps` times:  r = g - J1^T lambda (FP64, the entries of J1 evaluated on the fly from
 *   vm, va with the Alg. 1 formulas);  lambda += solve(r)   (solve = the transposed sweeps of sable_adjoint, in the
 *   precision of the kept factors).
 * sweeps = 0 is sable_adjoint.  vm, va = the vm, va returned by the last sable_solve; other arguments, layout and errors
 * as sable_adjoint (sweeps outside [0, 16]: INVALID_ARG).  All DEVICE pointers; asynchronous on the stream; for grids
 * above 3 413 buses the state part of the workspace is used as scratch (the kept factors stay intact). */
sable_status sable_adjoint_refined(sable_ctx* ctx, int32_t batch, const double* vm, const double* va,
                                   const double* g_va, const double* g_vm, int32_t sweeps, double* lam_p,
                                   double* lam_q, void* cuda_stream);

/* Host-buffer convenience wrappers: same semantics with HOST pointers (pinned memory for full copy speed); they copy in,
 * run on the context's device and copy out, synchronously.  The batch is cut into up to four chunks of whole scenario
 * groups, each on its own internal stream, so that the copies of one chunk overlap the kernels of the others.  The device
 * staging buffers are allocated at the first such call.  Used for the end-to-end measurement. */
sable_status sable_solve_host(sable_ctx* ctx, int32_t batch, const double* p_spec, const double* q_spec,
                              const double* v_set, const double* vm0, const double* va0, double tol,
                              int32_t max_it, double* vm, double* va, int32_t* iterations, uint8_t* converged,
                              double* final_norm);
sable_status sable_adjoint_host(sable_ctx* ctx, int32_t batch, const double* g_va, const double* g_vm,
                                double* lam_p, double* lam_q);

sable_status sable_get_info(const sable_ctx* ctx, sable_info* info);
const char*  sable_last_error(const sable_ctx* ctx);   /* ctx may be NULL: message of the last failed sable_create */
void         sable_destroy(sable_ctx* ctx);

/* Number of kernel launches the library has enqueued on this context since creation (for bench accounting). */
int64_t      sable_launch_count(const sable_ctx* ctx);

/* ---- debug / parity exports (used by tests; not part of the public surface) -------------------------------- */

/* Template queries (HOST out arrays; pass NULL to skip one).  Sizes come from sable_get_info.
 *   node_bus[n_node]      bus index of node p (nodes are in elimination order, grouped by level)
 *   node_level[n_node]
 *   pair_ptr[n_node+1]    pairs owned by node m are [pair_ptr[m], pair_ptr[m+1]); pair p = {U(m,j), L(j,m)}
 *   pair_col[n_pair]      node j of pair p (j > m)
 *   pair_in_j[n_pair]     1 if the pair is structurally present in J1, 0 if pure fill
 *   term_ptr[n_pair+1], term_a[n_term], term_b[n_term]   pair target p = (m,j) subtracts, for each term t,
 *                         L(m,k) U(k,j) and L(j,k) U(k,m) with term_a[t] = pair (k,m), term_b[t] = pair (k,j)
 *   dterm_ptr[n_node+1], dterm[n_pair]   diagonal target m subtracts L(m,k) U(k,m) for each pair dterm[t] = (k,m) */
sable_status sable_debug_pattern(const sable_ctx* ctx, int32_t* node_bus, int32_t* node_level, int32_t* pair_ptr,
                                 int32_t* pair_col, uint8_t* pair_in_j, int32_t* term_ptr, int32_t* term_a,
                                 int32_t* term_b, int32_t* dterm_ptr, int32_t* dterm);

/* Mismatch at a given state (DEVICE pointers, [batch][n_bus]): f_p[i] = P_i - P_spec,i (0 at slack),
 * f_q[i] = Q_i - Q_spec,i (0 off PQ), norm[b] = ||F1||_inf. */
sable_status sable_debug_mismatch(sable_ctx* ctx, int32_t batch, const double* p_spec, const double* q_spec,
                                  const double* vm, const double* va, double* f_p, double* f_q, double* norm,
                                  void* cuda_stream);

/* Jacobian blocks at a given state, written by the library's fill code in its padded block layout
 * (DEVICE out, doubles): diag[batch][n_node][4] = [dP/dth, dP/dVm, dQ/dth, dQ/dVm] of node m w.r.t. itself;
 * pairs[batch][n_pair][8] = block J1(m,j) (4 values, same order) followed by block J1(j,m).
 * Padded entries (V-column / Q-row of a PV node) are 0, except dQ/dVm = 1 on a PV diagonal. */
sable_status sable_debug_jacobian(sable_ctx* ctx, int32_t batch, const double* vm, const double* va,
                                  double* diag, double* pairs, void* cuda_stream);

/* One linear solve with the library's refactor + triangular solves at a given state:
 * transpose = 0: J1(V) x = rhs;  1: J1(V)^T x = rhs.  rhs_p/rhs_q and x_p/x_q are [batch][n_bus] DEVICE arrays
 * holding the theta/P component and the Vm/Q component per bus. */
sable_status sable_debug_linear_solve(sable_ctx* ctx, int32_t batch, const double* vm, const double* va,
                                      const double* rhs_p, const double* rhs_q, int32_t transpose,
                                      double* x_p, double* x_q, void* cuda_stream);

/* Per-stage times in the default workspace layout: runs the fused kernel's own stage routines one stage per launch
 * (mismatch + norm + decision + Jacobian fill / refactor + triangular solves + update) for three Newton iterations from the
 * flat start on the given batch (DEVICE pointers, [batch][n_bus]) and returns the mean CUDA-event time of each launch in ms
 * (HOST out).  Synchronous; overwrites the workspace, so kept factors are gone afterwards. */
sable_status sable_debug_stage_times(sable_ctx* ctx, int32_t batch, const double* p_spec, const double* q_spec,
                                     const double* v_set, double* ms_mismatch_fill, double* ms_factor_solve, void* cuda_stream);

/* Per-phase cycle counters of CTA 0 of the fused kernel, accumulated since the last call (then reset).  Only when
 * the context was created with tune.timing = 1 (else SABLE_ERR_STATE); the HBM-placement kernels
 * carry the counters only when the library is built with -DSABLE_TIMING_ALL (they cost registers there).  out[4 l + 0 / 2] = cycles
 * in the accumulate (factor + forward) / backward phase of elimination level l; out[4 L] = cycles in decision +
 * output; out[4 L + 1] = loop trips; out[4 L + 2] = refill + init; out[4 L + 3] = mismatch + norm; L = n_level;
 * n = entries wanted, at most 4 L + 4 (HOST out). */
sable_status sable_debug_timing(sable_ctx* ctx, uint64_t* out, int32_t n);

/* ---- the allocation-free entry point -------------------------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it):
 * the Step-2 recovery of sable_recover (PAPER.md:80 eq. 5, :95-99 eq. 9; S = V o conj(Y_bus V)) WITHOUT a context.
 * It calls no cudaMalloc, cudaFree or allocating library routine: the kernel's scratch (the voltages in rectangular form,
 * 16 bytes per bus and scenario) lives in one file-scope __device__ array of SABLE_STATIC_SCRATCH_BYTES that every GPU
 * loading the library holds until exit (csrc/sable_static.cu).
 *   n_bus, batch          batch * n_bus * 16 must not exceed SABLE_STATIC_SCRATCH_BYTES (524 288 voltages: e.g. 56 scenarios of
 *                         9 241 buses), else INVALID_ARG with a message that names the limit; batch = 0 only does the one-time
 *                         set-up for the current device (look-up of the array's address) -- do that before a graph capture
 *   row_ptr [n_bus+1], col_idx, y_re, y_im   Y_bus in CSR form, DEVICE pointers, read as given: any column order, duplicates
 *                         add up, indices must be valid (they cannot be checked without a copy)
 *   vm, va [batch][n_bus] DEVICE in;   p_inj, q_inj [batch][n_bus] DEVICE out: calculated net injections at every bus
 *   cuda_stream           cudaStream_t of the CURRENT device; the call only enqueues one kernel
 *   errbuf, errbuf_len    optional HOST buffer for the message of a failed call (may be NULL / 0)
 * Every call shares the one array: calls that overlap on the GPU (different streams, or different host threads) RACE on it and
 * must be serialised by the caller.  The array keeps the last call's contents; nothing in it has to start at zero (each
 * CTA writes its slice before reading it).  Errors: INVALID_ARG, CUDA. */
#define SABLE_STATIC_SCRATCH_BYTES (8u << 20)
sable_status sable_injections_static(int32_t n_bus, int32_t batch, const int32_t* row_ptr, const int32_t* col_idx,
                                     const double* y_re, const double* y_im, const double* vm, const double* va,
                                     double* p_inj, double* q_inj, void* cuda_stream, char* errbuf, int32_t errbuf_len);

#ifdef __cplusplus
}
#endif
#endif /* SABLE_H */

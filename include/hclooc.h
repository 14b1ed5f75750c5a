/* hclooc.h -- C ABI of libhclooc_b200: out-of-core FP64 matrix multiplication on one NVIDIA B200.
 *
 * The operation is the paper's MMOOC (arXiv 1808.05056; citations are PAPER.md:<line>):
 *
 *     C = alpha * A * B + beta * C        A is M x K, B is K x N, C is M x N, FP64   (:180, :275)
 *
 * with A, B and C resident in (pinned) host memory and the device restricted to a stated memory
 * budget (:277 "dMemSize", :289).  The library cuts A into horizontal slices, B into vertical slices
 * and C into blocks (:289, Figure 3 :281), streams them through device buffers on separate
 * host-to-device, compute and device-to-host CUDA streams synchronised with events (:291, :303-313),
 * and runs a hand-written sm_100a FP64 tile kernel per step (the "in-core DGEMM" of :308).
 *
 * Conventions for every function
 *   - Storage is ROW-MAJOR; leading dimensions are in ELEMENTS (doubles).  hclooc_dgemm is the paper's untransposed
 *     operation (:180); transposed operands and the other level-3 routines the paper names as future work (:412) have their
 *     own entry points below (hclooc_dgemm_t, hclooc_dsyrk, hclooc_dsyr2k, hclooc_dtrsm[_side], hclooc_dpotrf, hclooc_dgetrf).
 *   - All functions return an int status: 0 = success; a NEGATIVE value -k means the k-th argument
 *     (1-based, in the order of the C prototype) is invalid (LAPACK "info" convention); POSITIVE
 *     values are the HCLOOC_ERR_* codes below.  Nothing aborts and nothing throws across this ABI.
 *   - "host" pointers must be page-locked (hclooc_host_alloc / hclooc_host_register / cudaHostAlloc)
 *     and "device" pointers must come from hclMalloc / cudaMalloc on the current device.  There is no
 *     pageable or CPU fallback.
 *   - The library never takes ownership of caller memory.
 */
#ifndef HCLOOC_H
#define HCLOOC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ------------------------------------------------------------------ status codes */
#define HCLOOC_OK               0
#define HCLOOC_ERR_BUDGET       1   /* device budget below the minimum working set of the planner   */
#define HCLOOC_ERR_NOT_PINNED   2   /* A, B or C is pageable host memory (no silent fallback)       */
#define HCLOOC_ERR_CUDA         3   /* a CUDA call failed; see hclooc_last_cuda_error()             */
#define HCLOOC_ERR_NOMEM        4   /* device or host allocation failed                             */
#define HCLOOC_ERR_ALIGN        5   /* device operand not 16-byte aligned / odd leading dimension   */
#define HCLOOC_ERR_INTERNAL     6   /* planner/executor invariant violated (a bug)                  */
#define HCLOOC_ERR_NOALLOC_LIMIT 7  /* hclDgemmNoAlloc: shape beyond what its static scratch array serves */

/* ------------------------------------------------------------------ handles */
typedef struct hclooc_ctx hclooc_ctx;   /* opaque: device, streams, events, workspace              */
typedef void* hclStream;                /* a cudaStream_t (the paper's hclStream, :144)            */
typedef void* hclEvent;                 /* a cudaEvent_t  (the paper's hclEvent,  :146)            */

/* copy direction, the paper's enum Direction {H2D, D2H} (:136) */
#define HCL_H2D 0
#define HCL_D2H 1
/* op(X) of hclooc_dgemm_t: X as stored, or its transpose */
#define HCL_OP_N 0
#define HCL_OP_T 1

/* ------------------------------------------------------------------ the plan (hclMatrixPartitioner, :186, :289)
 * Loop structure:  for p < kpanels:  for j < w:  for i < h:  one step computes the C block
 * (rows i*mb .., cols j*nb ..) with the K panel p (k0 = p*kb):   c_ij = alpha*a_i*b_j + beta'*c_ij   (:308)
 * where beta' = beta for p == 0 and 1 afterwards.  Step index idx = i + h*(j + w*p) (:191 for p = 0).
 * Rows are visited in serpentine order (down the even columns of blocks, up the odd ones) so the A slices
 * still resident at the end of a column are reused by the next one instead of being uploaded again.
 * Edge slices are ragged (ceil division; the paper only treats equal slices).                       */
typedef struct hclooc_plan_t {
    int64_t  M, N, K;
    int64_t  mb, nb, kb;          /* rows of an A slice, columns of a B slice, depth of a K panel   */
    int64_t  h, w, kpanels;       /* ceil(M/mb), ceil(N/nb), ceil(K/kb)                             */
    int64_t  n_steps;             /* h * w * kpanels                                                */
    int32_t  n_sets;              /* C block device buffers, round-robin by step (the paper has 2)  */
    int32_t  n_bbuf;              /* B slice device buffers (1 = paper's single buffer, 2 = prefetch) */
    int32_t  beta_nonzero;        /* C blocks are uploaded only when 1 (or for K panels p > 0)      */
    int32_t  scale_only;          /* alpha == 0 or K == 0: C = beta*C, A and B never referenced     */
    int32_t  ksplit;              /* CTAs per cluster sharing one tile's K range in the kernel (1, 2, 4), or -1:
                                     every step is one persistent stream-K launch that fills the GPU by itself */
    int32_t  n_abuf;              /* A slice device buffers: an LRU cache keyed by (row slice, K panel) */
    int64_t  lda_dev, ldb_dev, ldc_dev;  /* leading dimensions of the device buffers (elements)    */
    uint64_t bytes_a_buf, bytes_b_buf, bytes_c_buf;   /* one buffer of each kind                   */
    uint64_t workspace_bytes;     /* n_bbuf*b + n_abuf*a + n_sets*c + n_scratch*bytes_scratch, <= the budget */
    uint64_t bytes_h2d, bytes_d2h;/* exactly what the executor enqueues over the host link          */
    uint64_t n_copies_h2d, n_copies_d2h;
    double   flops;               /* 2*M*N*K (:368)                                                 */
    double   t_flop_s, t_link_s, t_model_s;  /* cost model terms used to pick this plan             */
    int32_t  n_scratch;           /* stream-K scratch buffers (ksplit == -1): one per compute stream used       */
    int32_t  c_on_device;         /* 1: C lives in device memory: its block copies are device-to-device and are not
                                     counted in bytes_h2d / bytes_d2h (host-link bytes); 2: the result is written to device
                                     memory but the INITIAL C (the uploads of K panel 0) is read from a host matrix, which
                                     counts (a resident panel of hclooc_dpotrf / hclooc_dtrsm filled by the pipeline itself) */
    uint64_t bytes_scratch;       /* one of them (partial-tile slots + counters)                                */
    int32_t  direct;              /* 1 = DIRECT mode: no device buffer at all -- one launch of the tile kernel whose TMA
                                     loads read the A and B tiles straight from the (mapped) pinned host matrices and whose
                                     epilogue reads and writes C in host memory.  Every tile streams over the host link
                                     (bytes_h2d counts what the tiles read: A ceil(N/128)/direct_cn times, B ceil(M/128)/direct_cm
                                     times), so it only wins where the staged pipeline is bound by per-copy latency:
                                     small problems under small budgets (BASELINE config 1).  h = w = n_steps = 1.     */
    int32_t  direct_cm, direct_cn; /* direct mode: the launch runs clusters of direct_cm x direct_cn CTAs (neighbouring
                                     tiles) that share their loads by TMA multicast -- A is read ceil(ceil(N/128)/direct_cn)
                                     times and B ceil(ceil(M/128)/direct_cm) times; 4 x 4 (one 16-CTA cluster) makes
                                     config 1's traffic the compulsory minimum                                      */
    int32_t  tri;                 /* hclooc_dsyrk: 1 / 2 = only the lower / upper triangle of C is referenced; the schedule has no
                                     step for a block that lies wholly in the other triangle, and bytes_* / n_copies_* are
                                     those of the schedule (set by the executor; the planner leaves tri = 0)           */
    int32_t  resident;            /* != 0: the RESIDENT schedule ran (host matrices that fit the budget; resident.cu): A, B and C have
                                     device copies (lda_dev / ldb_dev / ldc_dev; bytes_a_buf / bytes_b_buf are the whole matrices and
                                     workspace_bytes also counts the M x ldc_dev copy of C), A and B go up in `kpanels` K panels of kb
                                     with whole-C kernels behind them, and from panel resident - 1 on C is finished in h row blocks
                                     of mb (w = 1): one launch over the remaining panels, dC += beta * C0 from a ring of n_sets
                                     staging buffers of bytes_c_buf, download.  n_steps = (resident - 1) + h DGEMM launches        */
    int32_t  trans;               /* hclooc_dgemm_t: bit 0 = A is stored K x M, bit 1 = B is stored N x K.  The device
                                     slices keep the stored layout: an A slice is then kb x mb (lda_dev >= mb), a B
                                     slice nb x kb (ldb_dev >= kb), and the tile kernel reads them transposed       */
} hclooc_plan_t;

/* Plan only (pure host arithmetic, needs no GPU).  alpha_zero != 0 plans the scale-only pass.
 * Errors: -1..-3 negative dimension, -7 NULL out, HCLOOC_ERR_BUDGET.                               */
int hclooc_plan(int64_t M, int64_t N, int64_t K, int beta_nonzero, int alpha_zero,
                size_t device_budget_bytes, hclooc_plan_t* out);
/* Same, saying where A, B and C live: 0 = pinned host memory (what hclooc_plan assumes), 1 = all three in
 * device memory: the in-core case (:130, :368) -- nothing is staged, the plan is one step over the caller's
 * matrices (h = w = 1, no buffers, no traffic).  hclooc_dgemm_ex picks this from the pointers it is given
 * (device operands that are not 16-byte aligned with even leading dimensions are staged like host ones);
 * 2 = A and B in pinned host memory, C in device memory (the nsteps mode below): C blocks move device to
 * device, so they cost no host-link time and are not counted in bytes_h2d / bytes_d2h;
 * 3 = as 0, and the device can address the host matrices as they are (mapped pinned memory, 16-byte aligned, even
 * leading dimensions): the cost model may then pick the DIRECT mode (plan.direct) when it beats every staged plan;
 * 4 = as 3 but direct mode is forced (tests, experiments); 5 = as 2, but the initial C is read from a host matrix
 * (plan.c_on_device = 2: the C uploads of K panel 0 count as link traffic).  -8: NULL out. */
int hclooc_plan_ex(int64_t M, int64_t N, int64_t K, int beta_nonzero, int alpha_zero,
                   size_t device_budget_bytes, int operands_on_device, hclooc_plan_t* out);

/* Same for hclooc_dgemm_t (declared below): transa / transb = HCL_OP_N (0) or HCL_OP_T (1) say which operands are stored
 * transposed; their device slices keep the stored layout (plan.trans), which changes buffer sizes and leading dimensions
 * and makes thin row slices of a transposed A expensive to upload (rows of mb doubles).  -8 / -9: transa / transb invalid,
 * -10: NULL out.                                                                                                       */
int hclooc_plan_trans(int64_t M, int64_t N, int64_t K, int beta_nonzero, int alpha_zero, size_t device_budget_bytes,
                      int operands_on_device, int transa, int transb, hclooc_plan_t* out);

/* The RESIDENT schedule's shape for a call whose A, B and C fit the budget (pure host arithmetic; what hclooc_dgemm consults after
 * planning the slices): applies = 1 if hclooc_dgemm would run it -- M, N, K >= 1024 and M*N*K >= 8e9 (small calls are latency bound:
 * direct mode and graph replay own them), the device copies + stream-K scratch + staging ring within the budget, at least two K
 * panels, and the schedule's estimate t_model_s below 0.985 * t_slice_model_s (pass the slice plan's plan.t_model_s; <= 0 skips the
 * comparison); HCLOOC_RESIDENT=0 / 1 in the environment forces the answer where the schedule fits at all.  The shape is filled
 * whenever it fits: h row blocks of mb rows, `npanels` K panels [panel_k0[p], panel_k0[p] + panel_kk[p]) graded from 256 or 512
 * columns up to kb, phase 2 from panel p_switch on, `ring` staging buffers for the initial C (0 when beta == 0), workspace_bytes.
 * Errors: -1..-3 non-positive dimension, -7 NULL out.                                                                         */
#define HCLOOC_RESIDENT_MAX_PANELS 128
typedef struct hclooc_resident_plan_t {
    int32_t  applies, ring;
    int64_t  mb, h, kb, npanels, p_switch;
    int64_t  lda_dev, ldb_dev, ldc_dev;
    uint64_t workspace_bytes;
    double   t_flop_s, t_link_s, t_model_s;
    int64_t  panel_k0[HCLOOC_RESIDENT_MAX_PANELS], panel_kk[HCLOOC_RESIDENT_MAX_PANELS];
} hclooc_resident_plan_t;
int hclooc_plan_resident(int64_t M, int64_t N, int64_t K, int beta_nonzero, size_t device_budget_bytes, double t_slice_model_s,
                         hclooc_resident_plan_t* out);
/* The resident schedule as the exact list of operations hclooc_dgemm enqueues for it, in host issue order (hclooc_op_t, declared
 * below with the pipeline's schedule).  Streams: 0 = uploads, 1 = downloads, 2.. = compute (phase 2 alternates between 2 and 3 when
 * n_compute >= 2).  Device buffers: 0 = the copy of A, 1 = of B, 2 = of C, 3 + s = staging slot s of the initial C.  Per kind:
 * H2D_A / H2D_B: K panel [k0, k0 + kk) (all rows of A / those rows of B); GEMM: dC[r0 : r0 + nr, :] = alpha * dA[r0.., k0 : k0 + kk] *
 * dB[k0.., :] + beta * dC[...]; H2D_C: host C rows [r0, r0 + nr) -> staging slot `buf`; AXPY: dC[r0.., :] += beta_call * slot `buf`;
 * D2H_C: dC rows -> host C rows.  Events: panel p uploaded = p; C0 block r uploaded = npanels + r; slot of block r free again =
 * npanels + h + r; row block r finished = npanels + 2h + r; phase 1 finished = npanels + 3h.  The tests run a vector-clock hazard
 * check over this list without a GPU.  Errors: -1 plan NULL or inconsistent with M, -2..-4 dimensions, -6 n_compute < 1, -9 NULL.  */
struct hclooc_op_t;
int hclooc_resident_schedule(const hclooc_resident_plan_t* plan, int64_t M, int64_t N, int64_t K, int beta_nonzero, int n_compute,
                             struct hclooc_op_t* ops, size_t max_ops, size_t* n_ops);

/* The paper's own rule, kept for reference and tests (:289, worked example :301): EQUAL slices only,
 * working set K*nb + 2*mb*K + 2*mb*nb <= budget_elements, least host-to-device traffic
 * w*M*K + K*N + M*N; ties: fewest steps, then smallest h.  Returns HCLOOC_ERR_BUDGET if nothing fits. */
int hclMatrixPartitioner(int64_t M, int64_t N, int64_t K, int64_t budget_elements, int64_t* h, int64_t* w);

/* ------------------------------------------------------------------ the schedule (S2-S7 as a list of stream operations)
 * hclooc_schedule() expands a plan into the exact sequence of operations the executor enqueues, in
 * host issue order: copies, kernels, and the event records/waits that order them across streams
 * (the paper's five event families eA, rA, rB, eC, rC, :187-188, :291, :311).  The executor issues this
 * very list, so tests can check coverage, byte counts and hazard freedom without a GPU.            */
#define HCLOOC_OP_H2D_A   0   /* S(a_i)  :306  host A[r0:r0+nr, c0:c0+nc] -> device buffer `buf`            */
#define HCLOOC_OP_H2D_B   1   /* S(b_j)  :305  host B[r0.., c0..] -> rows dev_r0.. of device buffer `buf`   */
#define HCLOOC_OP_H2D_C   2   /* S(c_ij) :307  host C[r0.., c0..] -> device buffer `buf`                    */
#define HCLOOC_OP_GEMM    3   /* DGEMM   :308  buf3(C) = alpha*buf(A)*buf2(B) + beta*buf3(C); nr x nc x kk  */
#define HCLOOC_OP_D2H_C   4   /* R(c_ij) :309  device buffer `buf` -> host C[r0.., c0..]                    */
#define HCLOOC_OP_WAIT    5   /* stream waits for event (hclWaitEvent, :116)                              */
#define HCLOOC_OP_RECORD  6   /* event recorded in stream (Rec(x), :311)                                  */
#define HCLOOC_OP_AXPY    7   /* resident schedule only: dC[r0.., :] += beta * staging buffer `buf`       */
/* streams: 0 = H2D copy stream, 1 = D2H copy stream, 2 + c = compute stream c.
 * buffers: A slice buffer a = a; C block buffer c = n_abuf + c; B slice buffer b = n_abuf + n_sets + b.
 * events:  c = uploads of the step using C buffer c arrived (rA/rC); n_sets + c = its kernel finished (eA);
 *          2*n_sets + c = C buffer c stored on the host (eC); 3*n_sets + b = B buffer b received (rB);
 *          3*n_sets + n_bbuf + b = every kernel of the column that read B buffer b finished;
 *          3*n_sets + 2*n_bbuf + 2*a + (0|1) = the kernels that read A buffer a finished (readers alternate). */
typedef struct hclooc_op_t {
    int32_t kind, stream, event;
    int32_t buf, buf2, buf3;
    int64_t r0, nr, c0, nc;       /* region of the host matrix (GEMM: nr x nc output block)          */
    int64_t dev_r0;               /* first row inside the device buffer (B prefetch chunks)          */
    int64_t k0, kk;               /* GEMM: K panel                                                    */
    int64_t step;                 /* idx = i + h*(j + w*p)                                            */
    double  beta;                 /* GEMM: effective beta of this step                                */
} hclooc_op_t;

/* Writes up to max_ops operations to ops (may be NULL to only count) and the total count to *n_ops.
 * n_compute = number of compute streams the executor will round-robin over (>= 1).                  */
int hclooc_schedule(const hclooc_plan_t* plan, int n_compute, hclooc_op_t* ops, size_t max_ops, size_t* n_ops);

/* ------------------------------------------------------------------ statistics of one call */
typedef struct hclooc_stats {
    hclooc_plan_t plan;
    uint64_t bytes_h2d, bytes_d2h;      /* counted at enqueue time; equal plan.bytes_*              */
    uint64_t n_kernels, n_copies_h2d, n_copies_d2h;
    double   t_total_s;                 /* wall time of the call, entry to return (:368 "including transfers") */
    double   t_enqueue_s;               /* host time spent enqueueing                               */
} hclooc_stats;

/* ------------------------------------------------------------------ context
 * device: CUDA ordinal.  d_workspace/workspace_bytes: caller-owned device memory (e.g. a PyTorch
 * tensor) the context carves all its buffers from, or NULL/0 to let the library cudaMalloc (and grow)
 * its own.  stream_h2d / stream_d2h: caller-owned cudaStream_t or NULL for library-owned.
 * compute_streams[n_compute]: caller-owned compute streams, or NULL/0 for 8 library-owned ones.    */
int hclooc_ctx_create(hclooc_ctx** ctx, int device, void* d_workspace, size_t workspace_bytes,
                      hclStream stream_h2d, hclStream stream_d2h, hclStream* compute_streams, int n_compute);
int hclooc_ctx_destroy(hclooc_ctx* ctx);

/* Tracing (debug aid): when enabled, the next hclooc_dgemm_ex calls on this context
 * bracket every copy and kernel with timing events; hclooc_ctx_get_trace returns, for the LAST call, one
 * record per operation with start/end in milliseconds relative to the first operation of that call.
 * ctx == NULL addresses the default context.  Tracing costs two event records per operation.       */
typedef struct hclooc_trace_rec {
    int32_t  kind, stream;        /* HCLOOC_OP_* and stream index as in hclooc_op_t                  */
    int64_t  step;
    uint64_t bytes;               /* bytes moved (copies) or 0                                        */
    double   flops;               /* 2*m*n*k (kernels) or 0                                           */
    double   t_start_ms, t_end_ms;
} hclooc_trace_rec;
int hclooc_ctx_set_trace(hclooc_ctx* ctx, int enable);
/* Direct mode (plan.direct) policy of this context: -1 = let the cost model choose (default), 0 = never (every call
 * is staged through device buffers), 1 = always when the operands allow it.  -2: mode outside {-1, 0, 1}.   */
int hclooc_ctx_set_direct(hclooc_ctx* ctx, int mode);
int hclooc_ctx_get_trace(hclooc_ctx* ctx, hclooc_trace_rec* recs, size_t max_recs, size_t* n_recs);
/* Calibrates the planner's cost model to THIS box: measures the host link of the context's device (256 MiB of pinned 64 MiB copies:
 * host->device alone, device->host alone, both at once; about 60 ms) and replaces the model's default rates -- those of the first
 * box probed, 55.5 / 51.5 / 88 GB/s; the boxes of a pool differ by 10 % -- for every later plan of the process (rates pinned by
 * the HCLOOC_*_GBPS environment variables stay).  The three outputs (nullable) receive the rates in GB/s.  ctx == NULL: default
 * context.  Errors: HCLOOC_ERR_CUDA (allocation or copy failed; the model is left as it was).                               */
int hclooc_calibrate_link(hclooc_ctx* ctx, double* h2d_GBps, double* d2h_GBps, double* duplex_GBps);
/* Debug shaker (the rule it exercises is PAPER.md:311: "data stored in device buffers is not overwritten until
 * kernel executions that operate on the data have completed").  jitter_seed != 0: every copy and kernel the library enqueues on this
 * context -- the DGEMM pipeline, the device phases of hclooc_dtrsm[_side] and hclooc_dpotrf -- is preceded, with probability 1/2,
 * by a spin kernel of random length (up to ~150 us) in its stream, so that the streams drift against each other differently in
 * every call.  poison != 0: a device buffer region is filled with NaN at the moment the schedule declares it free -- in front of
 * the upload that overwrites it (behind that upload's waits) and behind the download of a C block -- so that a reader the event
 * waits failed to order sees NaN instead of stale but plausible data.  A schedule that is race free gives the same results with
 * the shaker on (the parity tests run under it); CUDA-graph replay is off while it is on.  HCLOOC_DEBUG_JITTER=<seed> in the
 * environment switches both on for every context created afterwards.  poison == 2 additionally SABOTAGES the pipeline (its
 * upload stream skips every event wait): the tests use it to show that the shaker does turn a missing wait into wrong results.
 * Returns 0.                                                                                                                */
int hclooc_ctx_set_debug(hclooc_ctx* ctx, uint64_t jitter_seed, int poison);

/* ------------------------------------------------------------------ the operation
 * hclooc_dgemm: C = alpha*A*B + beta*C, synchronous: C is complete in host memory on return.
 *   A: M x K, lda >= K;  B: K x N, ldb >= N;  C: M x N, ldc >= N, updated IN PLACE; A, B read-only.
 *   A, B, C: pinned HOST pointers (the product path).  Device pointers are also accepted: if all three are
 *   device memory the call is in-core (one DGEMM on the caller's matrices, nothing staged) -- bench.py's
 *   HBM-resident `value` leg; a mix is staged through the workspace with device-to-device copies.  The call runs on the
 *   context's own non-blocking streams, which do not wait for work the caller has in flight on other streams: device operands
 *   must be COMPLETE (their producing copies / kernels synchronised) before they are handed over.
 *   device_budget_bytes bounds the sum of all device buffers the call uses (0 = all free HBM minus a
 *   1 GiB margin).  Uses a process-wide default context created on first use.
 *   beta == 0: C is never read (NaN/Inf in C are overwritten).  alpha == 0 or K == 0: A and B are not
 *   referenced, C = beta*C streamed through the device.  M == 0 or N == 0: returns 0, touches nothing.
 *   Schedules: slices of A, B and C through the buffers of a plan (hclooc_plan; the paper's pipeline, :182-271); DIRECT mode for
 *   small latency-bound calls (plan.direct); and, when A, B and C all FIT the budget and the cost model prefers it, the RESIDENT
 *   schedule (plan.resident: K streamed in panels behind the uploads, C finished row block by row block under its own downloads;
 *   HCLOOC_RESIDENT=0 / 1 in the environment forces the choice).  Floating-point results of different schedules agree within the
 *   1e-13 * D gate, not bit for bit (the order of summation over K differs); integer-valued data is exact under all of them.
 * Errors: -1/-2/-3 negative M/N/K; -5 A NULL; -6 lda < K; -7 B NULL; -8 ldb < N; -10 C NULL or C
 *   overlaps A or B; -11 ldc < N; HCLOOC_ERR_BUDGET; HCLOOC_ERR_NOT_PINNED; HCLOOC_ERR_NOMEM;
 *   HCLOOC_ERR_CUDA.  Validation errors leave C untouched; after HCLOOC_ERR_CUDA C is unspecified.  */
int hclooc_dgemm(int64_t M, int64_t N, int64_t K, double alpha, const double* A, int64_t lda,
                 const double* B, int64_t ldb, double beta, double* C, int64_t ldc,
                 size_t device_budget_bytes);

/* Same with an explicit context (NULL = default) and optional statistics (argument numbers in error
 * codes are those of hclooc_dgemm).  If the context has a caller-owned workspace the budget is
 * min(device_budget_bytes or workspace size, workspace size).                                      */
int hclooc_dgemm_ex(hclooc_ctx* ctx, int64_t M, int64_t N, int64_t K, double alpha, const double* A,
                    int64_t lda, const double* B, int64_t ldb, double beta, double* C, int64_t ldc,
                    size_t device_budget_bytes, hclooc_stats* stats_out);

/* Transposed operands (SURVEY 8(f) #3; the paper lists them as future work, :412):
 *     C = alpha * op(A) * op(B) + beta * C,   op(X) = X (HCL_OP_N) or X^T (HCL_OP_T)
 * op(A) is M x K and op(B) is K x N: with transa = HCL_OP_T, A is stored K x M (lda >= M); with transb = HCL_OP_T, B is
 * stored N x K (ldb >= K).  Nothing is transposed in memory: slices cross the link and sit in their device buffers in
 * the layout they are stored in, and the tile kernel reads them through tensor maps and fragment addressing made for
 * that layout (four variants of the same DMMA loop; the order of summation over k is that of hclooc_dgemm_ex, so the
 * result has the same bits as a call on written-out transposes).  Plan, schedule, events, direct mode and the in-core
 * case are those of hclooc_dgemm_ex.
 * Errors: as hclooc_dgemm_ex with the argument numbers of hclooc_dgemm (-6: lda too small for the STORED shape, ...),
 * plus -15 / -16: transa / transb is neither HCL_OP_N nor HCL_OP_T.                                                  */
int hclooc_dgemm_t(hclooc_ctx* ctx, int transa, int transb, int64_t M, int64_t N, int64_t K, double alpha,
                   const double* A, int64_t lda, const double* B, int64_t ldb, double beta, double* C, int64_t ldc,
                   size_t device_budget_bytes, hclooc_stats* stats_out);

/* Out-of-core DSYRK on the same path (SURVEY 8(f) #3: "other level-3 BLAS out of core"; the paper's future work, :412):
 *     C = alpha * A * A^T + beta * C   (trans = HCL_OP_N, A is N x K, lda >= K)
 *     C = alpha * A^T * A + beta * C   (trans = HCL_OP_T, A is K x N, lda >= N)
 * C is N x N symmetric and only its `uplo` triangle (HCL_UPLO_LOWER / HCL_UPLO_UPPER, diagonal included) is referenced: the
 * other triangle is bit-for-bit what it was on return.  It is one pass of the hclooc_dgemm_t pipeline with a triangle mask
 * (plan.tri): the schedule has no step for a block of C that lies wholly in the other triangle, the kernels skip such tiles
 * inside the blocks that cross the diagonal and store only their referenced elements, so about half the flops and half the
 * C traffic of the corresponding DGEMM are spent.  C blocks that cross the diagonal are uploaded
 * even when beta == 0 (their other-triangle part must come back unchanged); a NaN there is carried, never computed with.
 * alpha == 0 or K == 0: C = beta*C on the triangle, A not referenced.  stats (nullable) as hclooc_dgemm_ex.  Errors: -2 uplo, -3 trans, -4 N < 0, -5 K < 0, -7 A NULL, -8 lda too small, -10 C NULL or overlapping A,
 * -11 ldc < N, and the HCLOOC_ERR_* codes of hclooc_dgemm.                                                              */
#define HCL_UPLO_LOWER 0
#define HCL_UPLO_UPPER 1
int hclooc_dsyrk(hclooc_ctx* ctx, int uplo, int trans, int64_t N, int64_t K, double alpha, const double* A, int64_t lda,
                 double beta, double* C, int64_t ldc, size_t device_budget_bytes, hclooc_stats* stats_out);

/* Out-of-core DSYR2K, two masked passes of the same pipeline (the second accumulates with beta' = 1):
 *     C = alpha*A*B^T + alpha*B*A^T + beta*C   (trans = HCL_OP_N, A and B are N x K, lda, ldb >= K)
 *     C = alpha*A^T*B + alpha*B^T*A + beta*C   (trans = HCL_OP_T, A and B are K x N, lda, ldb >= N)
 * on the `uplo` triangle of the N x N matrix C; the other triangle keeps its bits.  Rounding: the first product is rounded
 * into C with beta*C, the second is then added (what the oracle's dsyr2k does).  stats: sums over the two passes.
 * Errors: -2 uplo, -3 trans, -4 N < 0, -5 K < 0, -7 A NULL, -8 lda, -9 B NULL, -10 ldb, -12 C NULL or overlapping A or B,
 * -13 ldc < N, and the HCLOOC_ERR_* codes.                                                                            */
int hclooc_dsyr2k(hclooc_ctx* ctx, int uplo, int trans, int64_t N, int64_t K, double alpha, const double* A, int64_t lda,
                  const double* B, int64_t ldb, double beta, double* C, int64_t ldc, size_t device_budget_bytes,
                  hclooc_stats* stats_out);

/* Out-of-core DTRSM, side = Left (the paper's future work, :412):  solve
 *     op(T) * X = alpha * B,   op(T) = T (trans = HCL_OP_N) or T^T (HCL_OP_T),
 * where T is the `uplo` triangle of the M x M matrix A (row-major, lda >= M; the other triangle is never read, nor is the
 * diagonal when diag = HCL_DIAG_UNIT) and B is M x N (ldb >= N); X overwrites B in place.  A and B are pinned host memory
 * (device memory is accepted too and staged the same way).  Blocked substitution: B is cut into block rows of NB <= 4096
 * rows (8192 where two such block rows fit in device memory; NB*NB*8 <= half the budget); a block row first receives  B_i <- alpha*B_i - op(T)[i, solved]*X[solved]  as ONE
 * out-of-core DGEMM through the hclooc_dgemm_t pipeline, then its diagonal block is solved in device memory: T_ii is
 * uploaded once, B_i streams through two column-chunk buffers on two streams, and inside a chunk 128-row triangles are
 * solved by a substitution kernel (one thread per column of B) with the tile kernel updating the rows still to be solved.
 * Rounding: substitution with the sums over k taken in blocked order; the result satisfies the elementwise residual bound
 * |alpha*B - op(T) X| <= gamma_(M+2) (|alpha B| + |op(T)||X|) of substitution in any order (G23), and is exact on
 * integer data with a +-1 diagonal.  alpha == 0: X = 0, A not referenced.  M == 0 or N == 0: nothing is done.
 * stats (nullable): byte / copy / kernel counts summed over the DGEMM calls and the diagonal phases; plan.mb = NB,
 * plan.nb = chunk width, plan.h = block rows, plan.flops = M*M*N, plan.workspace_bytes = the most device memory used.
 * Errors: -2 uplo, -3 trans, -4 diag, -5 M < 0, -6 N < 0, -8 A NULL, -9 lda < M, -10 B NULL or overlapping A,
 * -11 ldb < N; HCLOOC_ERR_BUDGET when not even a 32-row block fits; the HCLOOC_ERR_* codes of hclooc_dgemm.  A singular
 * T gives Inf / NaN as in the BLAS (no check).  Validation errors leave B untouched.
 * Experiment knobs (environment, read once): HCLOOC_TRSM_RESIDENT=0 staged mode only; HCLOOC_TRSM_NB_MAX=n block-row height;
 * HCLOOC_TRSM_CHUNKS / HCLOOC_TRSM_STREAMS column chunks and streams of the resident diagonal phase (default 8 / 2);
 * HCLOOC_TRSM_TIMING=1 prints the time of each block row's update and diagonal phase to stderr.                          */
#define HCL_DIAG_NONUNIT 0
#define HCL_DIAG_UNIT    1
int hclooc_dtrsm(hclooc_ctx* ctx, int uplo, int trans, int diag, int64_t M, int64_t N, double alpha, const double* A, int64_t lda,
                 double* B, int64_t ldb, size_t device_budget_bytes, hclooc_stats* stats_out);

/* The shape hclooc_dtrsm works in (pure host arithmetic, needs no GPU): *NB = rows of a block row (<= 4096, or <= 8192 in resident mode; NB*NB*8 <= half the
 * budget, a multiple of 128 -- of 32 below 128 -- or M itself), *chunk = columns of a staged column chunk (multiple of 64),
 * *resident = block rows kept in device memory (2, 1, or 0 = staged mode; always 0 unless library_owned: a context working in
 * caller-owned device memory allocates nothing), *device_bytes = what the diagonal phase holds (resident block rows + triangle
 * buffer, or triangle buffer + two chunk buffers); in resident mode a quarter of the budget at least is left to the DGEMM calls.
 * Errors: -1 M < 1, -2 N < 1, -5 NULL output, HCLOOC_ERR_BUDGET when not even a 32-row block with 64-column chunks fits.   */
int hclooc_dtrsm_plan(int64_t M, int64_t N, size_t device_budget_bytes, int library_owned, int64_t* NB, int64_t* chunk,
                      int* resident, uint64_t* device_bytes);

/* DTRSM with a side argument (BLAS order of arguments).  side = HCL_SIDE_LEFT is hclooc_dtrsm above (error codes then count
 * the arguments of THIS prototype).  side = HCL_SIDE_RIGHT solves
 *     X * op(T) = alpha * B,    T = the `uplo` triangle of the N x N matrix A (lda >= N),  B is M x N (ldb >= N), X overwrites B.
 * Every row of B is an independent system: the rows are cut into bands whose block columns (NB <= 4096 columns; the NB x NB
 * triangle and a band of one block column each take at most a quarter of the budget) sit in device memory one at a time; a
 * block column first receives  B_j <- alpha*B_j - X[:, solved] * op(T)[solved, j]  as one out-of-core DGEMM (C in device
 * memory), then its diagonal block is solved there by recursive halving down to 128-column blocks (one thread per row of B in
 * the block kernel).  When two whole block columns (M x NB, NB = 4096, 2048 or 1024) and two NB x NB blocks of T leave a quarter
 * of the budget to the DGEMM pipeline, the LOOK-AHEAD form runs instead (plan.n_sets = 2): block column j is solved in device
 * memory and downloaded in row chunks while the pipeline brings block column j+1 up with the update from the columns solved
 * before j; HCLOOC_TRSM_LOOKAHEAD=0 in the environment keeps the staged form.  Rounding and gate as hclooc_dtrsm (DESIGN.md
 * G23) with N in place of M; exact on integer data with a power-of-two diagonal.  alpha == 0: X = 0, A not referenced.
 * stats: plan.mb = band height (staged) / rows per chunk (look-ahead), plan.nb = NB, plan.flops = M*N*N.
 * Errors: -2 side, -3 uplo, -4 trans, -5 diag, -6 M < 0, -7 N < 0, -9 A NULL, -10 lda too small, -11 B NULL or overlapping A,
 * -12 ldb < N; HCLOOC_ERR_BUDGET when not even a 32-column block fits; the HCLOOC_ERR_* codes of hclooc_dgemm.             */
#define HCL_SIDE_LEFT  0
#define HCL_SIDE_RIGHT 1
int hclooc_dtrsm_side(hclooc_ctx* ctx, int side, int uplo, int trans, int diag, int64_t M, int64_t N, double alpha,
                      const double* A, int64_t lda, double* B, int64_t ldb, size_t device_budget_bytes, hclooc_stats* stats_out);

/* Out-of-core Cholesky factorization (DPOTRF; the paper's future work, :412: "out-of-core factorizations (LU, QR, Cholesky) that
 * use the out-of-core matrix-matrix multiplication (DGEMM) as a fundamental building block"):
 *     uplo = HCL_UPLO_LOWER:  A = L * L^T,  L overwrites the lower triangle of A;    HCL_UPLO_UPPER:  A = U^T * U,  U the upper one.
 * A is N x N, symmetric positive definite, row-major in pinned host memory (lda >= N); only its `uplo` triangle is read and
 * written, the other triangle keeps its bits.  Left-looking by panels of NB <= 4096 columns (rows, for the upper factor) with a
 * LOOK-AHEAD of one panel: two panels sit in device memory (at most half the budget: 2 * N * NB * 8 bytes).  While panel j is
 * factored there -- its diagonal block by recursive halving whose flops sit in tile-kernel launches (128 x 128 blocks by a one-CTA
 * kernel), the rest of the panel solved against it (X L_jj^T = P, the right-side DTRSM above) -- panel j+1 is uploaded and receives
 * the contribution of the panels before j as ONE out-of-core DGEMM with the triangle mask (hclooc_dsyrk's) streamed from the host;
 * panel j's own contribution then comes straight from device memory, and panel j goes back to the host beside all that.
 * *info (LAPACK): 0, or k > 0 when the leading minor of order k is not positive definite -- the factorization stops; the
 * panels before the one holding column k-1 are complete, that panel is left partly factored (as LAPACK leaves it undefined) and
 * the panels after it are unchanged.  The function still returns 0 then.
 * Rounding: the factor satisfies |A - L L^T| <= gamma_(N+2) |L||L^T| elementwise (any order of summation does, Higham thm 10.3;
 * DESIGN.md G24); exact on integer data whose factor is integer with a power-of-two diagonal.
 * stats (nullable): sums over the DGEMM calls and the panel copies; plan.nb (lower) / plan.mb (upper) = NB, plan.flops = N^3/3.
 * Errors: -2 uplo, -3 N < 0, -4 A NULL, -5 lda < N, -7 info NULL; HCLOOC_ERR_BUDGET when not even a 32-column panel fits half
 * the budget (N * 512 bytes); the HCLOOC_ERR_* codes of hclooc_dgemm.  Experiment knob: HCLOOC_POTRF_NB=n panel width.      */
int hclooc_dpotrf(hclooc_ctx* ctx, int uplo, int64_t N, double* A, int64_t lda, size_t device_budget_bytes,
                  int64_t* info, hclooc_stats* stats_out);
/* The panel width hclooc_dpotrf works with (pure host arithmetic) and the device bytes of its resident panel.
 * Errors: -1 N < 1, -3 NULL output, HCLOOC_ERR_BUDGET.                                                                      */
int hclooc_dpotrf_plan(int64_t N, size_t device_budget_bytes, int64_t* NB, uint64_t* panel_bytes);

/* Out-of-core LU factorization with partial pivoting (the paper's future work: "out-of-core factorizations (LU, QR,
 * Cholesky) that use the out-of-core matrix-matrix multiplication (DGEMM) as a fundamental building block", G27):
 *     P * A = L * U
 * A is M x N, row-major in PINNED HOST memory (lda >= N, in elements), overwritten in place by L (below the diagonal, unit diagonal
 * not stored, |l_ij| <= 1) and U (on and above it) -- LAPACK DGETRF's result for the row-major matrix, L in the FINAL row order.
 * ipiv: min(M, N) entries of HOST memory (pageable is fine), written: ipiv[j] = the row, 0-BASED (LAPACK: 1-based), exchanged with
 * row j at step j; the pivot of a column is its entry of largest magnitude from the diagonal down, the FIRST one on ties.
 * Left-looking over block columns of NB columns (hclooc_dgetrf_plan): a panel of all M rows stays in device memory while, for every
 * block column before it, it takes that block's interchanges, a device DTRSM against the block's unit lower triangle and one
 * out-of-core DGEMM (L streamed from the host, the panel in device memory); then its rows from the diagonal down are factored in
 * device memory (recursive halving: tile-kernel DGEMMs and DTRSMs; at the bottom a cooperative multi-CTA kernel that keeps a
 * panel of up to 128 columns in shared memory and pays one grid barrier per column).  The host matrix sees no row interchange until a final
 * pass brings every block column of L into the final order.  Look-ahead of one panel: the call starts ONE worker thread per panel
 * (joined before it returns) that drives the device factorization of panel j on a stream of its own while the calling thread drives the
 * out-of-core updates of panel j+1; three panels stay resident where they fit 7/8 of the budget, else two in 5/8 (knobs:
 * HCLOOC_GETRF_PANELS=2|3, HCLOOC_GETRF_LOOKAHEAD=0 factors in line).  Synchronous: returns with A and ipiv complete.
 * *info (LAPACK): 0, or j+1 > 0 for the first pivot u_jj that is exactly zero (the factorization is completed all the same; U is
 * singular).  The function still returns 0 then.  NaN in A: unspecified pivots.
 * Rounding: |P A - L U| <= gamma_n |L||U| elementwise, n = min(M, N) (Gaussian elimination in any order of operations, Higham
 * thm 9.3 / section 13.2); on data whose elimination is exact in FP64 the result is bit-identical to the unblocked definition.
 * stats (nullable): sums over the DGEMM calls and the panel copies; plan.nb = NB, plan.flops = M N^2 - N^3/3 (M >= N).
 * Errors: -2 M < 0 (or >= 2^31), -3 N, -4 A NULL, -5 lda < N, -6 ipiv NULL, -8 info NULL; HCLOOC_ERR_BUDGET when two 32-column
 * panels and their scratch do not fit 5/8 of the budget (about 2 * M * 256 bytes + 1/4 MiB); the HCLOOC_ERR_* codes of hclooc_dgemm.  Knob: HCLOOC_GETRF_NB=n.     */
int hclooc_dgetrf(hclooc_ctx* ctx, int64_t M, int64_t N, double* A, int64_t lda, int64_t* ipiv, size_t device_budget_bytes,
                  int64_t* info, hclooc_stats* stats_out);
/* The panel width hclooc_dgetrf works with (pure host arithmetic) and the device bytes it keeps for itself (two or three panels, two
 * diagonal blocks, scratch).  Errors: -1 M < 1, -2 N < 1, -4 NULL output, HCLOOC_ERR_BUDGET.                                 */
int hclooc_dgetrf_plan(int64_t M, int64_t N, size_t device_budget_bytes, int64_t* NB, uint64_t* reserved_bytes);
/* The device phase on its own: P A = L U of an M x N row-major matrix in DEVICE memory (16-byte aligned, lda even), in place, on
 * stream s.  ipiv (min(M, N) entries) and info are HOST memory.  NOT asynchronous: the host folds each panel's interchanges into
 * a permutation before the kernels that apply them are enqueued, so the call returns with the factorization complete; it
 * allocates (and frees) its scratch -- at most 64 MiB + 2 MiB of device memory, 1 MiB + 8 min(M, N) bytes of pinned host memory.
 * Errors: -1 M, -2 N, -3 dA NULL, -4 lda, -5 ipiv NULL, -6 info NULL; HCLOOC_ERR_ALIGN, HCLOOC_ERR_NOMEM, HCLOOC_ERR_CUDA.      */
int hclDgetrf(int64_t M, int64_t N, double* dA, int64_t lda, int64_t* ipiv, int64_t* info, hclStream s);

/* Out-of-core DTRMM and DSYMM (the paper's future work, :412: "full support for level-3 BLAS kernels"): the routines whose operand
 * is a TRIANGLE of a stored matrix.  The pipeline streams the stored matrix as it is and the tile kernel is told which part of
 * op(A) / op(B) counts: a tile runs only over the k blocks that can hold counted elements, and in the blocks that cross the
 * diagonal the rest is zeroed by a select -- the other triangle (and a unit diagonal) is never multiplied, NaN there is harmless.
 *   hclooc_dtrmm:  B := alpha * op(T) * B (side = HCL_SIDE_LEFT, T = the `uplo` triangle of the M x M matrix A) or
 *     B := alpha * B * op(T) (HCL_SIDE_RIGHT, A is N x N), B is M x N (ldb >= N), IN PLACE.  Left: one pass of the pipeline with C = B
 *     (a step reads device copies of its operands made before the first block of its column is stored; needs a budget that holds a
 *     16-column slice of B without K panels, else HCLOOC_ERR_BUDGET).  Right: B goes through the device in row bands (a band is copied
 *     up once, at most a quarter of the budget, and is the left operand of its own pass).  diag = HCL_DIAG_UNIT: the strict triangle
 *     multiplies and B itself enters as beta * C with beta = alpha.  alpha == 0: B = 0, A not referenced.
 *     Errors: -2 side, -3 uplo, -4 trans, -5 diag, -6 M < 0, -7 N < 0, -9 A NULL, -10 lda too small, -11 B NULL or overlapping A,
 *     -12 ldb < N, and the HCLOOC_ERR_* codes.  stats: plan of the (last) pass, byte / copy / kernel counts summed, plan.flops = M*N*n.
 *   hclooc_dsymm:  C := alpha * S * B + beta * C (HCL_SIDE_LEFT, S is M x M) or alpha * B * S + beta * C (HCL_SIDE_RIGHT, S is N x N), S the
 *     symmetric matrix whose `uplo` triangle is stored in A (the other triangle is never read), B and C M x N.  Two passes of the
 *     pipeline: the stored triangle, then its strict part read transposed with beta' = 1 (rounding: the first partial sum is rounded
 *     into C with beta*C, the second is added; within the gate of hclooc_dgemm, exact on integers).  alpha == 0: C = beta*C.
 *     Errors: -2 side, -3 uplo, -4 M < 0, -5 N < 0, -7 A NULL, -8 lda, -9 B NULL, -10 ldb < N, -12 C NULL or overlapping A or B,
 *     -13 ldc < N, and the HCLOOC_ERR_* codes.  stats: sums over the two passes, plan.flops = 2*M*N*n.                          */
int hclooc_dtrmm(hclooc_ctx* ctx, int side, int uplo, int trans, int diag, int64_t M, int64_t N, double alpha,
                 const double* A, int64_t lda, double* B, int64_t ldb, size_t device_budget_bytes, hclooc_stats* stats_out);
int hclooc_dsymm(hclooc_ctx* ctx, int side, int uplo, int64_t M, int64_t N, double alpha, const double* A, int64_t lda,
                 const double* B, int64_t ldb, double beta, double* C, int64_t ldc, size_t device_budget_bytes,
                 hclooc_stats* stats_out);

/* nsteps mode (:277-283): MMOOC as a subroutine of a blocked algorithm (SUMMA, HSUMMA) that updates the same C
 * `nsteps` times: C = alpha*A_p*B_p + beta_p*C for p = *step = 0 .. nsteps-1, one call per p.  C is uploaded once
 * at step 0 (if beta != 0), stays in device memory between the calls, and is downloaded once at the last step, so
 * every call moves only its A and B over the host link (the paper's listing of this logic is garbled, :245,
 * :259-263; this is its stated intent).  C (M x N, must fit the budget beside a working set) counts against
 * device_budget_bytes; host C is untouched until the last step.  *step is incremented on success (the caller
 * starts a sequence with *step = 0); a failed call ends the sequence and releases the device copy.
 * Errors as hclooc_dgemm, plus -13 nsteps < 1, -14 step NULL or outside [0, nsteps), -10 also when C, M, N or ldc
 * differ from the running sequence; HCLOOC_ERR_BUDGET when C does not fit.  stats as hclooc_dgemm_ex; the one
 * upload / download of C is added to the byte counts of the first / last call.                          */
int hclooc_dgemm_nsteps(hclooc_ctx* ctx, int64_t M, int64_t N, int64_t K, double alpha, const double* A,
                        int64_t lda, const double* B, int64_t ldb, double beta, double* C, int64_t ldc,
                        size_t device_budget_bytes, int nsteps, int* step, hclooc_stats* stats);

/* Multi-GPU (SURVEY 8(e); the paper's future work, :414): the row blocks of C are independent (:289, :293), so
 * G processes, one per GPU, each take a contiguous band of the rows of A and C and all of B, and call
 * hclooc_dgemm on their band -- no exchange step, no collective.  This returns the band of `rank`: the M rows
 * are cut into `world` near-equal bands whose sizes are multiples of `align` rows (128 = the kernel's tile
 * edge; 1 = any), the remainder going to the last non-empty band; trailing ranks may get rows = 0.
 * Errors: -1 M < 0, -2 world < 1, -3 rank outside [0, world), -4 align < 1, -5/-6 NULL.              */
int hclooc_shard_rows(int64_t M, int world, int rank, int64_t align, int64_t* row0, int64_t* rows);

/* The paper's own pipeline, Figure 2 (:182-271), written against the hcl* runtime calls below and kept for
 * comparison with the tuned scheduler: hclMatrixPartitioner's equal slices (h | M, w | N),
 * steps in column-major order, TWO round-robin streams, five event families (eA, rA, rB, eC, rC), double
 * buffered A slice and C block, a single B buffer reloaded un-overlapped at i == h-1; in-core (one upload,
 * one DGEMM, one download) when A, B and C fit device_budget_bytes together (:130, :368).  Same arguments,
 * result and error codes as hclooc_dgemm (M, N, K > 0 required: -1/-2/-3); allocates its device buffers with
 * hclMalloc per call (at most device_budget_bytes; 0 = free HBM minus 1 GiB).  stats (nullable): plan.h/w/mb/nb,
 * byte and copy counts, n_kernels; t_total_s runs from the first enqueue to both streams drained.        */
int hclooc_dgemm_fig2(int64_t M, int64_t N, int64_t K, double alpha, const double* A, int64_t lda,
                      const double* B, int64_t ldb, double beta, double* C, int64_t ldc,
                      size_t device_budget_bytes, hclooc_stats* stats);

/* ------------------------------------------------------------------ the runtime the paper abstracts (:109-116, :212)
 * CUDA only, plain functions (no virtual dispatch, cf. :164).                                      */
int hclMalloc(void** dptr, size_t bytes);                         /* :109  device memory            */
int hclFree(void* dptr);                                          /* :110                           */
int hclGetMemSize(int device, size_t* free_bytes);                /* :111  free device memory       */
int hclStreamCreate(hclStream* s);                                /* hclStreamFactory::create, :144 */
int hclStreamDestroy(hclStream s);
int hclEventDestroy(hclEvent e);
int hclMemcpy(void* dst, const void* src, size_t bytes, int dir);                         /* :112   */
/* Async calls take a stream and optionally create+record an event tied to the call (:140-146):
 * if ev != NULL and *ev == NULL a new event is created; the event is recorded after the operation. */
int hclMemcpyAsync(void* dst, const void* src, size_t bytes, int dir, hclStream s, hclEvent* ev);   /* :113 */
/* 2-D strided copy (rows x width_bytes, pitches in bytes): needed for row-major column slices; not in the paper. */
int hclMemcpy2DAsync(void* dst, size_t dpitch, const void* src, size_t spitch, size_t width_bytes,
                     size_t rows, int dir, hclStream s, hclEvent* ev);
/* In-core DGEMM on DEVICE pointers -- the tile kernel, one step of the pipeline (:212, :308):
 *   dC = alpha*dA*dB + beta*dC, row-major.  dA, dB, dC 16-byte aligned, lda/ldb/ldc even, else
 *   HCLOOC_ERR_ALIGN.  beta == 0: dC is not read.  K == 0 or alpha == 0: dC = beta*dC.              */
int hclDgemmAsync(int64_t M, int64_t N, int64_t K, double alpha, const double* dA, int64_t lda,
                  const double* dB, int64_t ldb, double beta, double* dC, int64_t ldc,
                  hclStream s, hclEvent* ev);
/* Same with the launch variant spelled out: HCL_DGEMM_AUTO (what hclDgemmAsync does: the persistent stream-K
 * kernel when the output has at least 148 tiles of 128 x 128, else one CTA -- or a cluster of 2 or 4 CTAs
 * splitting K -- per tile), 1 / 2 / 4 = that many CTAs per tile (what a pipeline step launches, plan.ksplit),
 * -1 = persistent stream-K; HCL_DGEMM_CLUSTER(cm, cn), cm, cn in {1, 2, 4} = the direct-mode kernel: clusters of
 * cm x cn neighbouring tiles sharing their A / B loads by TMA multicast (plan.direct_cm / direct_cn).  -14: unknown.  */
#define HCL_DGEMM_AUTO 0
#define HCL_DGEMM_CLUSTER(cm, cn) (100 + 10 * (cm) + (cn))
int hclDgemmAsyncEx(int64_t M, int64_t N, int64_t K, double alpha, const double* dA, int64_t lda,
                    const double* dB, int64_t ldb, double beta, double* dC, int64_t ldc,
                    hclStream s, hclEvent* ev, int variant);
/* Same on transposed device operands: dC = alpha*op(dA)*op(dB) + beta*dC with dA stored K x M when transa = HCL_OP_T
 * (lda >= M) and dB stored N x K when transb = HCL_OP_T (ldb >= K).  variant as hclDgemmAsyncEx.
 * -15 / -16: transa / transb invalid.                                                                              */
int hclDgemmAsyncT(int transa, int transb, int64_t M, int64_t N, int64_t K, double alpha, const double* dA, int64_t lda,
                   const double* dB, int64_t ldb, double beta, double* dC, int64_t ldc,
                   hclStream s, hclEvent* ev, int variant);
/* In-core DTRSM and DPOTRF on DEVICE pointers, asynchronous in stream s -- the device phases of hclooc_dtrsm[_side] and
 * hclooc_dpotrf as calls of their own (recursive halving down to 128 x 128 blocks: the flops sit in tile-kernel launches, the
 * blocks go to the substitution / factorization block kernels).  dA, dB 16-byte aligned, lda, ldb even, else HCLOOC_ERR_ALIGN.
 *   hclDtrsmAsync:  op(T) X = alpha B (side = HCL_SIDE_LEFT, T is M x M) or X op(T) = alpha B (HCL_SIDE_RIGHT, T is N x N), B is
 *     M x N and is overwritten by X.  Errors: -1 side, -2 uplo, -3 trans, -4 diag, -5 M < 0, -6 N < 0, -8 dA NULL, -9 lda, -10 dB
 *     NULL, -11 ldb < N.
 *   hclDpotrfAsync: the `uplo` triangle of the N x N matrix dA is overwritten by its Cholesky factor; *d_info (DEVICE memory,
 *     8 bytes) is zeroed and receives k > 0 if the leading minor of order k is not positive definite.  Errors: -1 uplo, -2 N < 0,
 *     -3 dA NULL, -4 lda < N, -5 d_info NULL.                                                                              */
int hclDtrsmAsync(int side, int uplo, int trans, int diag, int64_t M, int64_t N, double alpha, const double* dA, int64_t lda,
                  double* dB, int64_t ldb, hclStream s, hclEvent* ev);
int hclDpotrfAsync(int uplo, int64_t N, double* dA, int64_t lda, long long* d_info, hclStream s, hclEvent* ev);
/* The in-core DGEMM for callers that CANNOT ALLOCATE (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): dC = alpha*dA*dB + beta*dC on device pointers, row-major, the persistent stream-K kernel of hclDgemmAsyncEx(...,
 * variant -1) (the in-core kernel as a call of its own), asynchronous in stream s.  It calls no cudaMalloc,
 * cudaFree or allocating library routine, creates no event and no stream: the kernel's scratch (two partial 128 x 128 tiles per
 * persistent CTA and one counter per shared tile) is a static device array of HCL_NOALLOC_SCRATCH_BYTES (37.0 MiB) that every GPU
 * which loads the library holds until the process exits.
 *   Limits: M, N, K <= HCL_NOALLOC_MAX_DIM and ceil(M/128)*ceil(N/128) <= HCL_NOALLOC_MAX_TILES (what the kernel indexes with
 *   32-bit integers and the array has slots for: at most 148 persistent CTAs, 296 shared tiles); beyond them the call returns
 *   HCLOOC_ERR_NOALLOC_LIMIT and launches nothing.  No transposed operands, no event argument (record your own).
 *   EVERY call on a device shares the one array: two calls that overlap on the GPU (different streams, or graphs replayed
 *   concurrently) RACE on it and give wrong results -- keep the calls of a device in one stream or order them with events.  The
 *   array keeps the last call's contents; the call clears the counters it needs (a memset node in the stream), partial slots are
 *   written before they are read.
 *   dA, dB 16-byte aligned, lda, ldb even, else HCLOOC_ERR_ALIGN.  beta == 0: dC is not read.  K == 0 or alpha == 0: dC = beta*dC.
 *   Errors: -1..-3 negative dimension, -5 dA NULL, -6 lda < K, -7 dB NULL, -8 ldb < N, -10 dC NULL, -11 ldc < N,
 *   HCLOOC_ERR_NOALLOC_LIMIT, HCLOOC_ERR_ALIGN, HCLOOC_ERR_CUDA.                                                              */
#define HCL_NOALLOC_SCRATCH_BYTES 38798592
#define HCL_NOALLOC_MAX_DIM       2147483647LL
#define HCL_NOALLOC_MAX_TILES     1073741823LL
int hclDgemmNoAlloc(int64_t M, int64_t N, int64_t K, double alpha, const double* dA, int64_t lda,
                    const double* dB, int64_t ldb, double beta, double* dC, int64_t ldc, hclStream s);
size_t hclDgemmNoAllocScratchBytes(void);                        /* HCL_NOALLOC_SCRATCH_BYTES, as compiled           */
int hclWaitEvent(hclStream s, hclEvent e);                        /* :116  stream waits for event   */
int hclStreamSynchronize(hclStream s);                            /* :115                           */
int hclDeviceSynchronize(int device);                             /* :114                           */

/* ------------------------------------------------------------------ pinned host memory */
void* hclooc_host_alloc(size_t bytes);                 /* cudaHostAlloc; NULL on failure            */
int   hclooc_host_free(void* p);
int   hclooc_host_register(void* p, size_t bytes);     /* pin caller memory in place                */
int   hclooc_host_unregister(void* p);

/* ------------------------------------------------------------------ diagnostics */
const char* hclooc_strerror(int status);
int         hclooc_last_cuda_error(void);              /* last cudaError_t seen by this thread      */
const char* hclooc_version(void);
/* FP64 issue-rate probe of the current device: independent register chains of DMMA.8x8x4 (kind 0: mma.sync.m8n8k4.f64,
 * what the kernels use) or DFMA (kind 1), no memory traffic, ctas_per_sm x 256 threads per SM, launches repeated for
 * about `seconds`; writes the best launch in TFLOP/s.  The roofline denominator of DESIGN.md section 6 is this
 * measurement (python -m paper_1808_05056_b200.box_probe).  -1 kind, -2 ctas_per_sm outside 1..8, -3 seconds, -4 NULL. */
int hclooc_probe_fp64(int kind, int ctas_per_sm, double seconds, double* tflops);

#ifdef __cplusplus
}
#endif
#endif /* HCLOOC_H */

/*
 * casgd.h -- C ABI of libcasgd.so: one communication-avoiding SGD (CA-SGD) outer
 * iteration for generalized linear models on one NVIDIA B200 (sm_100a).
 *
 * Method: "Mixed-Precision Communication-Avoiding SGD for Generalized Linear
 * Models on GPUs" (arxiv/paper_2606_18463). Citations "PAPER.md:L<n>" are lines
 * of the paper's text; DESIGN.md lists every reading taken where the text is
 * silent or garbled. Scope: P = 1 (one GPU, Alg. 1 line 5's AllReduce is the
 * identity), Recipe C of Table 3 with r and u kept in FP32.
 *
 * Notation (sec. 3.1): A is the m x n data matrix (BF16), y the
 * m labels (FP32), x the n weights (FP32 master), b the mini-batch size, s the
 * number of inner steps, alpha = eta / b. One outer iteration takes sb = s*b row
 * indices I = I_0 u ... u I_{s-1} and computes (u = dL/dr = -delta):
 *
 *   Y   = A[I, :]                                   Alg. 1 line 2  (L113)   bit-exact
 *   r   = Y bf16(x)                                 line 3         (L114)   BF16 in, FP32 acc/out
 *   G   = Y Y^T   (blocks below the block diagonal) line 4         (L116)   BF16 in, FP32 acc/out
 *   z_j = r_j - alpha * sum_{k<j} G_{jk} u_k        lines 6-15     (L120-L132)   FP32
 *   u_j = l'(z_j, y_{I_j})                                                  FP32
 *   x  <- x - alpha * Y^T u                         lines 16-17    (L133-L135)   FP32 master
 *   bf16(x) refreshed for the next iteration        (L231)
 *
 * Conventions for every entry point
 *   - Pointers are DEVICE pointers on the context's GPU unless the parameter name
 *     ends in `_host`. Nothing is copied or retained beyond what is stated.
 *   - Every call returns a casgd_status. On failure casgd_last_error() gives a
 *     message. Nothing prints, throws or aborts. There is no CPU fallback: on a
 *     device that is not compute capability 10.x casgd_init returns CASGD_EARCH.
 *   - Calls that only enqueue work on the context's stream say "asynchronous";
 *     the others synchronise that stream before returning.
 *   - A context is not thread-safe; use one per host thread or lock around it.
 */
#ifndef CASGD_H
#define CASGD_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct casgd_ctx casgd_ctx; /* opaque; one per (A, y) dataset and CUDA device */

/* Loss family, sec. 2.1 (L) and L59 sec. 3.1 (delta = -dL/dr):
 *   LOGISTIC  L = log(1 + exp(-y r)),  u = -y / (1 + exp(y r)),  y in {-1, +1}
 *   LINEAR    L = (r - y)^2 / 2,       u = r - y
 *   POISSON   L = exp(r) - y r,        u = exp(r) - y,           y in {0, 1, 2, ...} */
typedef enum { CASGD_LOGISTIC = 0, CASGD_LINEAR = 1, CASGD_POISSON = 2 } casgd_loss_kind;

typedef enum {
    CASGD_OK = 0,
    CASGD_EINVAL = 1, /* bad argument (null, s < 1, b < 1, s*b > CASGD_MAX_SB, unknown loss/option, ...) */
    CASGD_ENOMEM = 2, /* device or host allocation failed */
    CASGD_ECUDA = 3,  /* a CUDA call or kernel failed; casgd_last_error() has the CUDA message */
    CASGD_EARCH = 4,  /* the current device is not sm_100 (B200) */
    CASGD_EINDEX = 5  /* a row index outside [0, m) was seen by a gather (sticky until casgd_sync) */
} casgd_status;

/* Largest s*b accepted: the paper's largest block, "sb <= 16384". */
#define CASGD_MAX_SB 16384

/* Create a context for the dataset (A, y).
 *   X_bf16  m x n BF16 bit patterns, row-major, row stride `ldx` elements (ldx >= n); all m * ldx elements
 *           must be readable. BORROWED for the context's lifetime: it is used in place when it can be
 *           (16-byte aligned base, ldx % 8 == 0); otherwise (e.g. n = 18, ldx = 18) the outer steps work on
 *           the library's own zero-padded copy, made during this call, and casgd_loss still streams the
 *           caller's (narrower) rows.
 *   m       rows, 1 <= m < 2^31 (every index buffer of this ABI is int32); n >= 1 columns.
 *   y       m FP32 labels (Table 1: labels are FP32 throughout). BORROWED.
 *   loss    a casgd_loss_kind.
 *   cuda_stream  a cudaStream_t (NULL = the legacy default stream). All work of this context is
 *           enqueued on it. BORROWED.
 * Synchronises `cuda_stream` if it had to copy X. The context allocates its workspaces lazily,
 * sized to the largest s*b seen. */
int casgd_init(casgd_ctx **out, const uint16_t *X_bf16, int64_t ldx, const float *y, int64_t m, int32_t n,
               int loss, void *cuda_stream);

/* One CA-SGD outer iteration, Algorithm 1 at P = 1. ASYNCHRONOUS.
 *   idx  s*b row indices in [0, m), int32; idx[j*b + i] is row i of mini-batch j. Any multiset is
 *        accepted (the paper samples with replacement, L111). An out-of-range index makes that
 *        row read as zeros with label 0 and raises the sticky CASGD_EINDEX flag.
 *   x    n FP32 master weights, updated in place: x <- x - (eta/b) Y^T u.
 * The BF16 shadow of x used by the margin (L231) is owned by the context. It is rebuilt from `x` at
 * the start of every casgd_outer_step / casgd_outer_steps* call (one n-element kernel per call) and kept
 * current by the fused update between the steps of a call, so a caller may change x, or pass another
 * x, between calls freely. */
int casgd_outer_step(casgd_ctx *c, const int32_t *idx, float *x, int32_t s, int32_t b, float eta);

/* n_steps consecutive outer iterations; step h uses idx[h*s*b .. (h+1)*s*b). ASYNCHRONOUS.
 * The same iterations as n_steps calls of casgd_outer_step without per-call launch cost: replayed from CUDA graphs of 64
 * steps, the remaining n_steps % 64 as one graph of that length (captured on first use and cached by length; an extension
 * of the paper's two CUDA graphs, L278), which pipeline consecutive iterations (CASGD_OPT_OVERLAP),
 * or, for steps small enough, run in ONE persistent launch (CASGD_OPT_MINI). Equal to the single-step calls bit for bit
 * where the same kernels run (CASGD_OPT_OVERLAP 0 and 1, the one-launch kernels), to FP32 rounding in the pipelined
 * graphs, whose margin is a kernel of its own. */
int casgd_outer_steps(casgd_ctx *c, const int32_t *idx, int64_t n_steps, float *x, int32_t s, int32_t b,
                      float eta);

/* n_steps outer iterations whose row indices are drawn ON THE DEVICE, i.i.d. uniformly with replacement as in
 * Alg. 1 line 1 -- no index upload. Counter-based: the indices of a step depend only on
 * (seed, step number, position), step h of this call being number first_step + h:
 *   index t:  counter = (t / 4, step mod 2^32, step div 2^32, 0xCA5D), key = (seed mod 2^32, seed div 2^32),
 *             w = Philox4x32-10(counter, key)[t mod 4],  idx = floor(w * m / 2^32)        (m < 2^31 by casgd_init)
 * (Salmon et al., SC'11). Otherwise exactly casgd_outer_steps on those indices. ASYNCHRONOUS. */
int casgd_outer_steps_sampled(casgd_ctx *c, int64_t n_steps, float *x, int32_t s, int32_t b, float eta, uint64_t seed,
                              uint64_t first_step);

/* The same through HOST buffers: copies idx_host (n_steps*s*b int32) and x_host (n FP32) to the
 * device, runs the steps, copies x back into x_host, and synchronises. Pinned host memory makes the
 * copies asynchronous with respect to the host but the call still returns only when x_host is valid; a call of one
 * step replays a one-step CUDA graph (one launch on a stream the host then waits for), and when both buffers are pinned
 * MAPPED host memory (cudaHostAlloc, torch's pin_memory()) and the call moves <= 64 KB of indices, one kernel reads them
 * in place and one writes x back -- no copy-engine round trips. A row index outside [0, m) is
 * reported here (CASGD_EINDEX; the row counts as zeros), as casgd_sync reports it for the asynchronous calls. */
int casgd_outer_steps_host(casgd_ctx *c, const int32_t *idx_host, int64_t n_steps, float *x_host, int32_t s,
                           int32_t b, float eta);

/* ---- P > 1 ranks, the paper's 1-D block-column partition (section 4.2; Alg. 1 line 5, L118) ----
 * Rank p creates its context on the column slab A[:, c0:c1] (n = c1 - c0, `ldx` the full row stride) with the FULL label
 * vector y, and owns the matching slab of x. One outer iteration is then
 *   casgd_step_local    gather Y_loc, G_loc = Y_loc Y_loc^T, r_loc = Y_loc x_loc (the context's Gram kernels), packed into
 *                       `payload_out`: casgd_payload_count(s, b) FP32 words, device memory, 16-byte aligned:
 *                         [ r_0 .. r_{sb-1} | block row 1 of G (b x b) | block row 2 (b x 2b) | .. | block row s-1 ]
 *                       entry (i, k), block(k) < block(i) = j, at  sb + b^2 j (j-1) / 2 + (i - j b) j b + k  -- r and the
 *                       strict block-lower part of G (L180), sb + b^2 s (s-1) / 2 words: half of Table 2's sb + (sb)^2
 *                       (L154), G being symmetric;
 *   the sum over ranks  (line 5) either by the caller -- e.g. an NCCL AllReduce of the payload (the paper's grouped
 *                       AllReduce, L276), then casgd_step_finish(payload_in = the reduced payload) -- or by
 *                       casgd_reduce_peers: one kernel of this library that reads every rank's payload (device pointers,
 *                       which may be peer-mapped memory of other GPUs reached over NVLink) and writes the sum, taken in
 *                       rank order so that all ranks hold identical bits, straight into the context's G and r (no staging
 *                       copy, no unpack pass); the caller orders it after every rank's casgd_step_local (events / a
 *                       barrier), then calls casgd_step_finish(payload_in = NULL);
 *   casgd_step_finish   the recurrence on the summed [r; G] (redundantly on every rank, L120-L132) and the update of this
 *                       rank's slab of x (L133-L135) and its shadow.
 * All ranks must pass the same idx, s, b, eta. ASYNCHRONOUS; errors as for casgd_outer_step. With P = 1 and
 * payload_in = the rank's own payload the three calls equal casgd_outer_step. */
int64_t casgd_payload_count(int32_t s, int32_t b);          /* -1 for arguments casgd_step_local would reject */
/* Payload buffers other PROCESSES can read (one process per GPU: each rank's casgd_reduce_peers reads every rank's
 * payload). casgd_payload_alloc makes a dedicated device allocation of `count` FP32 words (freed by casgd_payload_free);
 * casgd_ipc_export writes its 64-byte CUDA IPC handle to handle_host, which the caller sends to the other ranks by any
 * means; casgd_ipc_open maps a peer's handle into this process (a device pointer usable in casgd_reduce_peers' list;
 * over NVLink when the peer is another GPU), casgd_ipc_close unmaps it. */
int casgd_payload_alloc(int64_t count, float **payload_dev);
int casgd_payload_free(float *payload_dev);
int casgd_ipc_export(const float *payload_dev, void *handle_host /* 64 bytes */);
int casgd_ipc_open(const void *handle_host /* 64 bytes */, float **peer_payload_dev);
int casgd_ipc_close(float *peer_payload_dev);
int casgd_step_local(casgd_ctx *c, const int32_t *idx, const float *x, int32_t s, int32_t b, float *payload_out);
int casgd_reduce_peers(casgd_ctx *c, const float *const *peer_payloads_host, int32_t P, int32_t s, int32_t b);
int casgd_step_finish(casgd_ctx *c, float *x, int32_t s, int32_t b, float eta, const float *payload_in);

/* In-library baseline: one all-FP32 mini-batch SGD step, i.e. Alg. 1 with s = 1 and every
 * precision slot FP32 ("Recipe A", Table 3): x <- x - (eta/b) Y32^T l'(Y32 x, y_I), with
 * Y32 the exact FP32 widening of the BF16 rows. The first call allocates the m x n FP32 copy of A.
 * `idx` holds b indices; casgd_sgd_steps_fp32 runs n_steps of them. ASYNCHRONOUS. */
int casgd_sgd_step_fp32(casgd_ctx *c, const int32_t *idx, float *x, int32_t b, float eta);
int casgd_sgd_steps_fp32(casgd_ctx *c, const int32_t *idx, int64_t n_steps, float *x, int32_t b, float eta);

/* F(x) = (1/m) sum_i L(a_i^T x, y_i) over the whole dataset: BF16 A, FP32 x (the master,
 * not the shadow), FP32 margins and per-row losses, FP64 sum. Writes one double to *loss_host.
 * Synchronises. */
int casgd_loss(casgd_ctx *c, const float *x, double *loss_host);

/* The same F(x) WITHOUT A CONTEXT AND WITHOUT ANY ALLOCATION (csrc/loss_noalloc.cu), for callers that cannot call
 * cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid it. All pointers are DEVICE
 * pointers of the current device and stay the caller's: X_bf16 = m x n BF16 bit patterns with row stride ldx >= n
 * elements (any alignment; 16-byte-aligned rows take 16-byte loads), y = m FP32 labels, x = n FP32 weights,
 * result_dev = one double. loss = a casgd_loss_kind. ASYNCHRONOUS on cuda_stream (a cudaStream_t, or null).
 * The partial sums sit in a file-scope static __device__ array of 128 KB (one double per 256 rows) that every GPU loading
 * the library holds until exit: m <= 4,194,304, larger m returns CASGD_EINVAL (casgd_loss_noalloc_error() says why).
 * The first call on a device resolves the array's device address (cudaGetSymbolAddress; set-up, not an allocation) --
 * make it once outside a capture. Every call on a device shares the array: calls that overlap on the GPU (other
 * streams, concurrent graph replays) race; calls on one stream are ordered. Nothing has to start at zero (every slot a
 * call reads it has written). The summation order depends on (m, n) only: the same bits on every call. */
int casgd_loss_noalloc(const uint16_t *X_bf16, int64_t ldx, const float *y, int64_t m, int32_t n, int loss, const float *x,
                       double *result_dev, void *cuda_stream);
/* The calling thread's last casgd_loss_noalloc error message ("" after a successful call). */
const char *casgd_loss_noalloc_error(void);

/* Kept for compatibility: the shadow is rebuilt from x at the start of every outer-step call anyway. */
int casgd_invalidate_shadow(casgd_ctx *c);

/* Wait for the context's stream; returns CASGD_EINDEX (and clears the flag) if any gather since the
 * last casgd_sync saw an out-of-range index, CASGD_ECUDA if the stream failed. */
int casgd_sync(casgd_ctx *c);

/* Intermediates of the LAST outer step (casgd_outer_step, or the last step of casgd_outer_steps),
 * copied to HOST memory `dst_host`; synchronises. Layouts (sb = s*b of that step):
 *   CASGD_DBG_Y    sb x n  BF16 bits (uint16), packed row-major         (the gathered rows)
 *   CASGD_DBG_YLAB sb      FP32                                         (y_I)
 *   CASGD_DBG_G    sb x sb FP32 packed row-major. Valid entries: G[i][k] with block(k) < block(i)
 *                  always; every k <= i when CASGD_OPT_GRAM_FULL_LOWER is set. The rest is unspecified.
 *   CASGD_DBG_R    sb FP32   CASGD_DBG_Z sb FP32   CASGD_DBG_U sb FP32
 *   CASGD_DBG_XBF  n  BF16 bits: the shadow AFTER the step (bf16 of the updated x)
 *   CASGD_DBG_XSNAP  n FP32: with CASGD_OPT_SNAPSHOT, x as it entered the LAST step of the last CUDA graph replayed -- the
 *                  FP32 bits that step started from, so that a test can check it against the oracle element by element
 *   CASGD_DBG_GUARDS  1 int64: every per-step workspace (Y, y_I, G, r, z, u) sits between two 1 KB guard bands of a known
 *                  pattern; this is the number of guard bytes that no longer hold it (0 = no kernel wrote past a workspace)
 *   CASGD_DBG_STAMPS  64 x 8 x 2 uint64: with CASGD_OPT_STAMPS, {first-CTA start, last-CTA end} in %globaltimer ns of
 *                  stage g (CASGD_STAGE_*) of step h of the last graph casgd_outer_steps replayed, at [h][g][0..1];
 *                  {~0, 0} where a stage did not run
 * dst_bytes must equal the size implied above, else CASGD_EINVAL. */
typedef enum {
    CASGD_DBG_Y = 0, CASGD_DBG_YLAB = 1, CASGD_DBG_G = 2, CASGD_DBG_R = 3, CASGD_DBG_Z = 4,
    CASGD_DBG_U = 5, CASGD_DBG_XBF = 6, CASGD_DBG_STAMPS = 7, CASGD_DBG_GUARDS = 8, CASGD_DBG_XSNAP = 9
} casgd_debug_what;
int casgd_debug_export(casgd_ctx *c, int what, void *dst_host, int64_t dst_bytes);

/* Options (all default 0 unless stated).
 *   CASGD_OPT_GRAM_IMPL        0 = choose by a cost model (default), 1 = plain FP32-FMA CUDA-core kernel (bring-up
 *                              reference, same BF16 inputs and FP32 accumulation), 2 = tcgen05 kernel with 128 x 128
 *                              tiles, one CTA each, 3 / 4 = tcgen05 kernel on CTA pairs (cta_group::2) with
 *                              256 x 256 / 256 x 512 tiles (large shapes: fewer operand bytes per flop), 5 = gather and
 *                              Gram in ONE kernel, one CTA per 128 x 128 tile, rows pulled straight from A into the
 *                              swizzled operand layout (n <= 64 only; what 0 picks there).
 *   CASGD_OPT_GRAM_FULL_LOWER  1 = also compute the tiles on the block diagonal, so that the whole lower
 *                              triangle of CASGD_DBG_G is valid (the recurrence never reads them).
 *   CASGD_OPT_PROFILE          1 = record CUDA events around each stage of casgd_outer_step(s) (disables
 *                              graph replay); read with casgd_stage_times.
 *   CASGD_OPT_NO_GRAPH         1 = casgd_outer_steps launches kernels directly instead of replaying a graph.
 *   CASGD_OPT_GRAM_KSPLIT      0 = the tcgen05 Gram kernel chooses how many slices to cut K (= n) into so that
 *                              few-tile shapes still fill the GPU; k in [1, 64] forces k slices.
 *   CASGD_OPT_RECURRENCE_IMPL  0 = choose by the size of the strict block-lower G (default), 1 = the one-CTA
 *                              kernel, 2 = the grid-wide kernel (one CTA per SM, cooperative launch, u through
 *                              L2), 3 = the cluster kernel (one 16-CTA cluster, u through distributed shared
 *                              memory, G by plain loads; needs b % 4 == 0, else falls through to 2), 4 = the
 *                              streaming cluster kernel (same cluster, G through a cp.async.bulk shared-memory
 *                              ring; needs b % 4 == 0 and b <= 128, else falls through to 3), 5 = the chain-CTA
 *                              cluster kernel (blocks of 8..64 rows, b % 4 == 0, s*b <= 4096: the dependent chain on
 *                              ONE CTA, the older part of every sum from 15 helper CTAs; else falls through to 4).
 *   CASGD_OPT_NO_FUSED_UPDATE  1 = the outer update always runs as its own kernel. Default 0: for small steps
 *                              (at most 136 KB of Y per CTA of the cluster, 2048 columns) the streaming recurrence kernel's cluster does
 *                              g = Y^T u, the update of x and the shadow itself, right after the chain.
 *   CASGD_OPT_STAMPS           1 = every kernel of an outer step records when its first CTA started working (after its
 *                              programmatic-dependent-launch wait) and when its last CTA finished, in %globaltimer
 *                              nanoseconds; casgd_stage_times then returns, for the four step stages, the sum over
 *                              launches of (last end - first start) -- measured INSIDE the CUDA-graph replays that
 *                              casgd_outer_steps runs (unlike CASGD_OPT_PROFILE, which launches directly). Setting the
 *                              option (to 0 or 1) clears the totals.
 *   CASGD_OPT_OVERLAP          how the CUDA graphs of casgd_outer_steps schedule consecutive outer iterations (three Y and
 *                              two G stages): 0 = kernels strictly in sequence; 1 = a step that has a gather kernel
 *                              gathers the NEXT step's rows (Alg. 1 line 2 of iteration t + 1 needs no result of
 *                              iteration t) on a side branch, beside its own recurrence and update; 2 (default) =
 *                              pipelined: G(t+1) = Y Y^T needs no result of iteration t either, so the Gram of iteration
 *                              t + 1 runs on a branch of its own (on all but CASGD_OPT_CHAIN_SMS SMs) beside margin ->
 *                              recurrence -> update of iteration t, and the gather of iteration t + 2 beside that
 *                              recurrence; the margin r = Y x_bf, which does need x(t+1), is then a kernel of its own
 *                              (CASGD_STAGE_MARGIN) instead of extra B-operand rows of the Gram. Single-step calls run
 *                              the sequential kernels on the whole chip in every mode.
 *   CASGD_OPT_CHAIN_SMS        SMs left to the margin / recurrence / update chain in the pipelined schedule (the Gram and
 *                              gather kernels are sized for the rest). 0 (default) = 44, or 56 for steps of at least
 *                              16 MB of rows (measured).
 *   CASGD_OPT_MARGIN_SPLIT     0 (default) = Recipe C of Table 3: x enters the margin r = Y x as its BF16
 *                              shadow (L231, "two BF16 input conversions"). 1 = the margin sees the FP32 MASTER: rows 1
 *                              and 2 of the shadow buffer carry the BF16 residues of x (hi + lo + lo2 == x exactly), the
 *                              fused margin sums three accumulator columns, and the stand-alone margin kernel reads x
 *                              itself -- with A stored in BF16 this is Recipe B (u_A = b, every compute slot f): BF16 x
 *                              BF16 products are exact in FP32, so G and g are already what FP32 compute gives. Removes
 *                              the x half of Eq. 8's 2 u_16 term (L229) at no extra MMA.
 *   CASGD_OPT_MINI             1 (default) = steps small enough for one SM -- two stages of Y, the packed strict
 *                              block-lower G and the vectors within one CTA's shared memory, s*b <= 128, a Gram of at
 *                              most 460K multiply-adds: e.g. n = 64, s*b = 64; at s = 1 a step of <= 32 KB of rows (any
 *                              size for rows of <= 128 bytes), s*b <= 512 -- run ALL the iterations of a
 *                              casgd_outer_step(s) call in ONE persistent one-CTA launch (gather with the next
 *                              iteration's rows in flight, mma.sync Gram, recurrence, update, x resident in shared
 *                              memory), unless a kernel was asked for (CASGD_OPT_GRAM_IMPL, _RECURRENCE_IMPL,
 *                              _NO_FUSED_UPDATE, _GRAM_FULL_LOWER, _PROFILE); and s = 1 steps of more than 4 KB with
 *                              rows of >= 128 bytes, b <= 256, run them in one persistent launch of one thread-block
 *                              cluster that splits the columns
 *                              (s1_cluster.cu). 0 = always the kernel-per-stage path. 2 = the one-CTA launch whenever the
 *                              step FITS it (s*b <= 512, n <= 2048, shared memory), measured crossovers ignored: for
 *                              tests and for measuring those crossovers. 3 = likewise the cluster kernel whenever an
 *                              s = 1 step fits it.
 *   CASGD_OPT_SNAPSHOT         1 = the graphs of casgd_outer_steps copy x aside before their last step (CASGD_DBG_XSNAP):
 *                              test support, one n-element kernel per graph.
 *   CASGD_OPT_LOSS_IMPL        0 = casgd_loss streams A through per-warp cp.async.bulk shared-memory rings
 *                              (default; n <= 8192), 1 = the plain 16-byte-load kernel. */
typedef enum {
    CASGD_OPT_GRAM_IMPL = 0, CASGD_OPT_GRAM_FULL_LOWER = 1, CASGD_OPT_PROFILE = 2, CASGD_OPT_NO_GRAPH = 3,
    CASGD_OPT_GRAM_KSPLIT = 4, CASGD_OPT_RECURRENCE_IMPL = 5, CASGD_OPT_LOSS_IMPL = 6, CASGD_OPT_NO_FUSED_UPDATE = 7,
    CASGD_OPT_STAMPS = 8, CASGD_OPT_OVERLAP = 9, CASGD_OPT_CHAIN_SMS = 10, CASGD_OPT_MARGIN_SPLIT = 11, CASGD_OPT_MINI = 12, CASGD_OPT_SNAPSHOT = 13
} casgd_option;
int casgd_set_option(casgd_ctx *c, int option, int64_t value);

/* Stages of an outer step (plus shadow rebuilds = OTHER, and casgd_loss), for casgd_stage_times. MARGIN has launches of
 * its own only in the pipelined schedule (CASGD_OPT_OVERLAP = 2); otherwise r comes out of the Gram kernel. */
typedef enum {
    CASGD_STAGE_GATHER = 0, CASGD_STAGE_GRAM = 1, CASGD_STAGE_RECURRENCE = 2, CASGD_STAGE_GRADIENT = 3,
    CASGD_STAGE_MARGIN = 4, CASGD_STAGE_OTHER = 5, CASGD_STAGE_LOSS = 6, CASGD_NUM_STAGES = 7
} casgd_stage;

/* With CASGD_OPT_PROFILE set: total device milliseconds and launch counts per stage accumulated since
 * the option was set (or since the last call with reset != 0). ms_host and launches_host each hold
 * CASGD_NUM_STAGES entries. Synchronises. */
int casgd_stage_times(casgd_ctx *c, double *ms_host, int64_t *launches_host, int reset);

/* Number of kernels this context has launched (graph replays count their kernel nodes). */
int64_t casgd_launch_count(const casgd_ctx *c);

/* Message for the last non-OK status returned on this context ("" if none). Owned by the context. */
const char *casgd_last_error(const casgd_ctx *c);

/* Free everything the context owns (never X_bf16, y, idx, x). Synchronises. NULL is allowed. */
void casgd_destroy(casgd_ctx *c);

/* Library version string, and the SM architecture the kernels were compiled for ("sm_100a"). */
const char *casgd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CASGD_H */

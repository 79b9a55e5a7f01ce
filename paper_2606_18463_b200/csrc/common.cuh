// common.cuh -- shared declarations of libcasgd.so (device helpers, context, launch prototypes).
// Notation follows the paper (arxiv/paper_2606_18463): A, y, x, Y, G, r, z, u, b, s, alpha = eta/b.
#pragma once

#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>

#include "../../include/casgd.h"

namespace casgd {

constexpr int kTile = 128;            // Gram tile edge (rows of Y per tcgen05 operand tile)

// Device-side indirection block: lets kernels baked into a CUDA graph follow a base pointer
// that changes between replays (casgd_outer_steps).
struct StepParams {
    const int32_t *idx;   // first index of the current replay
    float *x;             // master weights
};

// ---------------------------------------------------------------- device math ---

__device__ __forceinline__ float bf16_bits_to_f32(uint16_t h) { return __uint_as_float(((uint32_t)h) << 16); }
__device__ __forceinline__ float bf16lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }

__device__ __forceinline__ uint16_t f32_to_bf16_bits_rn(float f)
{
    return __bfloat16_as_ushort(__float2bfloat16_rn(f));
}

// The BF16 view of x the margin reads. Row 0 of the [16 x ldxb] shadow buffer is bf16_rne(x). With
// CASGD_OPT_MARGIN_SPLIT (split_ld = ldxb, else 0) rows 1 and 2 carry the BF16 residues lo = bf16(x - hi) and
// lo2 = bf16(x - hi - lo): hi + lo + lo2 == x exactly (3 x 8 significand bits), every BF16 x BF16 product is exact
// in FP32, so the three accumulator columns of the fused margin sum to Y x with x the FP32 MASTER: the 2 u_16
// input-conversion term of Eq. 8 (L229) loses its x half at no extra MMA (the B operand has 16 rows anyway).
__device__ __forceinline__ void store_shadow(uint16_t *xbf, int32_t split_ld, int col, float xn)
{
    const __nv_bfloat16 hi = __float2bfloat16_rn(xn);
    xbf[col] = __bfloat16_as_ushort(hi);
    if (split_ld) {
        const float r1 = xn - __bfloat162float(hi);
        const __nv_bfloat16 lo = __float2bfloat16_rn(r1);
        xbf[split_ld + col] = __bfloat16_as_ushort(lo);
        xbf[2 * split_ld + col] = __bfloat16_as_ushort(__float2bfloat16_rn(r1 - __bfloat162float(lo)));
    }
}

// u = dL/dr = -delta. Accurate expf (not __expf): Poisson amplifies margin error by e^z.
template <int LOSS>
__device__ __forceinline__ float lprime(float z, float y)
{
    if (LOSS == CASGD_LOGISTIC) {
        float t = y * z;
        float e = expf(-fabsf(t));                   // in (0, 1]
        float sig_neg = (t >= 0.f) ? e / (1.f + e) : 1.f / (1.f + e);   // 1 / (1 + e^{t})
        return -y * sig_neg;
    } else if (LOSS == CASGD_LINEAR) {
        return z - y;
    } else {
        return expf(z) - y;
    }
}

__device__ __forceinline__ float lprime_rt(int loss, float z, float y)
{
    return loss == CASGD_LOGISTIC ? lprime<CASGD_LOGISTIC>(z, y)
         : loss == CASGD_LINEAR  ? lprime<CASGD_LINEAR>(z, y)
                                 : lprime<CASGD_POISSON>(z, y);
}

// log(1 + e) for e in [0, 1] as 2 atanh(w), w = e / (2 + e) in [0, 1/3]: the odd series up to w^15 (the next term
// is < 2e-9 of the result), relative error a few ulp for every e -- log1pf's accuracy at half its instructions (the
// narrow-row loss kernel is issue-bound).
__device__ __forceinline__ float log1p_unit(float e)
{
    const float w = __fdividef(e, 2.f + e), w2 = w * w;
    float p = 1.f / 15.f;
    p = fmaf(p, w2, 1.f / 13.f);
    p = fmaf(p, w2, 1.f / 11.f);
    p = fmaf(p, w2, 1.f / 9.f);
    p = fmaf(p, w2, 1.f / 7.f);
    p = fmaf(p, w2, 1.f / 5.f);
    p = fmaf(p, w2, 1.f / 3.f);
    p = p * w2;
    return 2.f * fmaf(w, p, w);
}

// L(r, y) in FP32; logistic as max(-t, 0) + log1p(exp(-|t|)).
__device__ __forceinline__ float loss_value_rt(int loss, float r, float y)
{
    if (loss == CASGD_LOGISTIC) {
        float t = y * r;
        return fmaxf(-t, 0.f) + log1p_unit(expf(-fabsf(t)));
    } else if (loss == CASGD_LINEAR) {
        float d = r - y;
        return 0.5f * d * d;
    }
    return expf(r) - y * r;
}

__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// dot of 8 BF16 (one 16-byte vector) with 8 FP32
__device__ __forceinline__ float dot8(const uint4 &a, const float4 &x0, const float4 &x1, float acc)
{
    acc = fmaf(bf16lo(a.x), x0.x, acc);
    acc = fmaf(bf16hi(a.x), x0.y, acc);
    acc = fmaf(bf16lo(a.y), x0.z, acc);
    acc = fmaf(bf16hi(a.y), x0.w, acc);
    acc = fmaf(bf16lo(a.z), x1.x, acc);
    acc = fmaf(bf16hi(a.z), x1.y, acc);
    acc = fmaf(bf16lo(a.w), x1.z, acc);
    acc = fmaf(bf16hi(a.w), x1.w, acc);
    return acc;
}

// dot of 8 BF16 with 8 BF16 (two 16-byte vectors), FP32 accumulation
__device__ __forceinline__ float dot8_bf16(const uint4 &a, const uint4 &x, float acc)
{
    acc = fmaf(bf16lo(a.x), bf16lo(x.x), acc); acc = fmaf(bf16hi(a.x), bf16hi(x.x), acc);
    acc = fmaf(bf16lo(a.y), bf16lo(x.y), acc); acc = fmaf(bf16hi(a.y), bf16hi(x.y), acc);
    acc = fmaf(bf16lo(a.z), bf16lo(x.z), acc); acc = fmaf(bf16hi(a.z), bf16hi(x.z), acc);
    acc = fmaf(bf16lo(a.w), bf16lo(x.w), acc); acc = fmaf(bf16hi(a.w), bf16hi(x.w), acc);
    return acc;
}

__device__ __forceinline__ uint4 ldg_nc_v4(const void *p)
{
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

// ------------------------------------------------- programmatic dependent launch ---
// The four kernels of an outer step are chained with programmatic stream serialisation: a kernel's CTAs are
// scheduled (and run their prologue) while the previous kernel drains, and block in pdl_wait() until it has
// completed and its writes are visible. Every kernel of the step path calls pdl_trigger() first thing and
// pdl_wait() before it touches anything another kernel of the chain writes or reads.
// IMPORTANT: what another kernel of the chain wrote must NOT be read through a `const T *__restrict__` pointer or
// __ldg: the compiler treats such data as read-only for the whole kernel and may hoist the load ABOVE pdl_wait()
// (seen: a gradient kernel summing the previous step's u). Such inputs are plain pointers, or go through ld_dep().
// A row index outside [0, m) was met: raise the context's flag. The flag lives in MAPPED PINNED HOST memory (the host
// reads it after a stream synchronize, no copy), so a plain store, not an atomic: every writer writes the same 1.
__device__ __forceinline__ void flag_index_error(int *err_flag) { *reinterpret_cast<volatile int *>(err_flag) = 1; }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ uint4 ld_dep_v4(const void *p)
{
    uint4 r;
    asm volatile("ld.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ float ld_dep(const float *p)
{
    float v;
    asm volatile("ld.global.f32 %0, [%1];" : "=f"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// ------------------------------------------------------------- in-graph stage stamps ---
// CASGD_OPT_STAMPS: every kernel of an outer step records when its first CTA got past pdl_wait() (atomicMin of
// %globaltimer) and when its last CTA finished (atomicMax) into a {t0, t1} slot of its (step, stage) -- the kernels run
// exactly as bench.py times them (CUDA-graph replay, programmatic dependent launch), unlike CASGD_OPT_PROFILE's direct
// launches. The slot pointer is a kernel argument baked into the graph (null = off). A launcher reads it from the
// thread-local g_stamp, which enqueue_step sets around each stage.
extern thread_local unsigned long long *g_stamp;
// Launch modifiers for the NEXT launch_pdl call(s) of this thread, set by the pipelined graph capture (casgd_api.cu):
// g_plain_launch: no programmatic-serialisation attribute (side-branch kernels must not become resident early: their
// waiting CTAs would hold the SMs the other branch needs); g_completion_event: record this event once all CTAs of the
// kernel have begun execution (cudaLaunchAttributeLaunchCompletionEvent; consumed by the launch).
extern thread_local bool g_plain_launch;
extern thread_local cudaEvent_t g_completion_event;
__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ void stamp_begin(unsigned long long *s)
{
    if (s && threadIdx.x == 0) atomicMin(s, globaltimer_ns());
}
__device__ __forceinline__ void stamp_end(unsigned long long *s)      // by thread 0, after the CTA's last barrier
{
    if (s && threadIdx.x == 0) atomicMax(s + 1, globaltimer_ns());
}
__device__ __forceinline__ void stamp_end_warp(unsigned long long *s) // by every warp (kernels whose warps end on their own)
{
    if (s && (threadIdx.x & 31) == 0) atomicMax(s + 1, globaltimer_ns());
}

// cudaLaunchKernelEx with the programmatic-serialisation attribute (and a cluster dimension when cluster > 1).
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, int cluster,
                              Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[3];
    int na = 0;
    if (!g_plain_launch) {
        attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    if (g_completion_event) {
        attr[na].id = cudaLaunchAttributeLaunchCompletionEvent;
        attr[na].val.launchCompletionEvent.event = g_completion_event;
        attr[na].val.launchCompletionEvent.flags = 0;
        ++na;
        g_completion_event = nullptr;
    }
    if (cluster > 1) {
        attr[na].id = cudaLaunchAttributeClusterDimension;
        attr[na].val.clusterDim.x = (unsigned)cluster;
        attr[na].val.clusterDim.y = 1;
        attr[na].val.clusterDim.z = 1;
        ++na;
    }
    cfg.attrs = attr;
    cfg.numAttrs = na;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// Per-device kernel attributes (opt-in shared memory sizes, non-portable cluster sizes): set for the CURRENT device by
// casgd_init, every time -- they are per device, so a process with contexts on several GPUs needs them on each.
cudaError_t gather_configure();
cudaError_t gradient_configure();
cudaError_t gram_tc_configure();
cudaError_t gram_pair_configure();
cudaError_t loss_configure();
cudaError_t recurrence_configure();
cudaError_t recurrence_stream_configure();
cudaError_t recurrence_chain_configure();
cudaError_t mini_step_configure();
cudaError_t s1_cluster_configure();

// ------------------------------------------------------------ launch prototypes ---
// Every launcher enqueues on `st` and returns the number of kernels it launched.
// `ind`, when non-null, overrides idx / x with ind->idx + idx_off / ind->x (graph replay).

int launch_gather(cudaStream_t st, const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n,
                  const int32_t *idx, const StepParams *ind, int64_t idx_off, int32_t sb, uint16_t *Y, int32_t ldy,
                  float *yI, int *err_flag, int num_sms);

int launch_gram_simt(cudaStream_t st, const uint16_t *Y, int32_t ldy, int32_t n, int32_t sb, int32_t b,
                     const uint16_t *xbf, int32_t split_ld, float *G, int32_t ldg, float *r, int full_lower);

// Cross-SM state of the grid-wide recurrence kernel (recurrence.cu).
struct RecWorkspace {
    unsigned long long *utag;      // [nrep x CASGD_MAX_SB] {u value, epoch tag} words, zero at allocation
    int32_t nrep;                  // replicas of the tagged words (spreads the polling over L2 slices)
    unsigned *epoch;               // tag of the next launch (starts at 1); retired by the kernel itself
    unsigned *done;                // CTAs finished in the current launch (0 between launches)
    int32_t max_ctas;              // CTAs that can be co-resident (one per SM); 0 = grid kernel unavailable
    int32_t cluster;               // CTAs per cluster of the cluster kernel (16 or 8); 0 = unavailable
    int64_t grid_threshold_bytes;  // strict block-lower G at or above this size leaves the one-CTA kernel
    int32_t late_trigger;          // 1 = the streaming kernel releases its dependent kernel only when the chain is done
                                   // (a side-branch gather needs the SMs the dependent's waiting CTAs would hold)
    int32_t g_protected;           // 1 = G was stored with L2::evict_last (the pair Gram kernel): the streaming kernel's
                                   // loads of it, the only ones there are, carry evict_first
};
int recurrence_cluster_size();
int recurrence_max_coresident_ctas(int num_sms);
// impl: 0 = choose by size, 1 = one CTA, 2 = all SMs through L2, 3 = one cluster, G from L2 by plain loads,
// 4 = one cluster, G through a cp.async.bulk ring (recurrence_stream.cu). Returns kernels launched, or -1 on a launch error.
// `fu` (optional): the outer update of the same step (Alg. 1 lines 16-17), which the streaming cluster kernel can do
// itself when Y is small; recurrence_fuses_update() tells whether launch_recurrence will honour it for this shape
// (the caller then skips the gradient kernel).
struct FusedUpdate {
    const uint16_t *Y;
    int32_t ldy, n;
    float *x;
    const StepParams *ind;
    uint16_t *xbf;
    int32_t split_ld;              // CASGD_OPT_MARGIN_SPLIT: row stride of the shadow buffer (0 = row 0 only)
    float *r_fused;                // non-null: the kernel also computes r = Y x_bf (Alg. 1 line 3) for its own rows first
};
bool recurrence_fuses_update(int32_t s, int32_t b, int32_t ldg, int32_t ldy, const RecWorkspace &ws, int impl);
int recurrence_kernel_choice(int32_t s, int32_t b, int32_t ldg, const RecWorkspace &ws, int impl, bool fused);
int launch_recurrence(cudaStream_t st, const float *G, int32_t ldg, const float *r, const float *yI, int32_t s,
                      int32_t b, float alpha, int loss, float *z, float *u, const RecWorkspace &ws, int impl,
                      const FusedUpdate *fu);

// recurrence_chain.cu: one cluster for blocks of <= 64 rows -- the chain on ONE CTA (no cluster crossing per hop), the
// older part of every row's sum from 15 helper CTAs. Kernel choice 5.
bool recurrence_chain_ok(int32_t s, int32_t b, int32_t ldg, int cluster);
bool recurrence_chain_fuses_update(int32_t s, int32_t b, int32_t ldy);
int launch_recurrence_chain(cudaStream_t st, const float *G, int32_t ldg, const float *r, const float *yI, int32_t s, int32_t b,
                            float alpha, int loss, float *z, float *u, const FusedUpdate *fu, int late_trigger);

// recurrence_stream.cu: one cluster, G streamed through a shared-memory ring, u through distributed shared memory.
bool recurrence_stream_ok(int32_t s, int32_t b, int32_t ldg, int cluster);
bool recurrence_stream_fuses_update(int32_t s, int32_t b, int32_t ldy, int cluster_max);
int launch_recurrence_stream(cudaStream_t st, const float *G, int32_t ldg, const float *r, const float *yI, int32_t s,
                             int32_t b, float alpha, int loss, float *z, float *u, int cluster, const FusedUpdate *fu,
                             int late_trigger);

struct GradWorkspace {
    float *partial;        // [row_splits x ldp] partial column sums
    int32_t ldp;
    unsigned *counters;    // one per column tile, zero between launches
    int32_t max_splits;
    int32_t num_sms;       // SMs of the context's device (grid sizing)
    int32_t split_ld;      // CASGD_OPT_MARGIN_SPLIT: row stride of the shadow buffer (0 = row 0 only)
};

int launch_gradient_bf16(cudaStream_t st, const uint16_t *Y, int32_t ldy, int32_t n, int32_t sb, const float *u,
                         float alpha, float *x, const StepParams *ind, uint16_t *xbf, const GradWorkspace &ws);

// s = 1 with wide rows: gather + margin + l' in one warp-per-row kernel (no Gram exists at s = 1); gradient.cu
// r = Y x_bf (Alg. 1 line 3) as a kernel of its own: the pipelined schedule computes G(t+1) before x(t+1) exists
// x32 / ind non-null (CASGD_OPT_MARGIN_SPLIT): the margin of the FP32 master itself, r = Y x
int launch_margin(cudaStream_t st, const uint16_t *Y, int32_t ldy, int32_t n, int32_t sb, const uint16_t *xbf, const float *x32,
                  const StepParams *ind, bool exact, float *r, int num_sms);

int launch_margin_s1(cudaStream_t st, const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n,
                     const int32_t *idx, const StepParams *ind, int64_t idx_off, int32_t b, int loss, const uint16_t *xbf,
                     int32_t split_ld, uint16_t *Y, int32_t ldy, float *yI, float *r, float *z, float *u, int *err_flag);

int launch_sgd32_step(cudaStream_t st, const float *A32, int64_t lda32, const float *y, int64_t m, int32_t n,
                      const int32_t *idx, int32_t b, float alpha, int loss, float *x, float *u, float *z,
                      int *err_flag, const GradWorkspace &ws);

int launch_loss(cudaStream_t st, const uint16_t *A, int64_t lda, const uint16_t *X, int64_t ldx, const float *y, int64_t m,
                int32_t n, int loss, const float *x, double *block_partials, int32_t max_blocks, double *result_dev,
                unsigned *done_counter, int impl, int num_sms);

int launch_sample_indices(cudaStream_t st, int32_t *idx, int64_t n_steps, int32_t sb, int64_t m, uint64_t seed,
                          uint64_t first_step);
int launch_snapshot(cudaStream_t st, const float *x, const StepParams *ind, int32_t n, float *dst);
int launch_shadow(cudaStream_t st, const float *x, const StepParams *ind, int32_t n, uint16_t *xbf, int32_t ldxb, int split);
int launch_widen(cudaStream_t st, const uint16_t *A, int64_t lda, int64_t m, int32_t n, float *A32, int64_t lda32, int num_sms);
int launch_repack(cudaStream_t st, const uint16_t *X, int64_t ldx, int64_t m, int32_t n, uint16_t *A, int64_t lda, int num_sms);
int launch_set_params(cudaStream_t st, StepParams *ind, const int32_t *idx, float *x);
int launch_stage_in(cudaStream_t st, const int32_t *idx_host, int64_t count, int32_t *idx_stage, const float *x_host, int32_t n,
                    float *x_stage, uint16_t *xbf, int32_t ldxb, int split);
int launch_stage_out(cudaStream_t st, const float *x_stage, int32_t n, float *x_host);
// slots: [nslots][2] {min start, max end} in %globaltimer ns, slot = 8 * step + stage; accum_ns / count: [8]
int launch_stamp_collect(cudaStream_t st, unsigned long long *slots, int nslots, unsigned long long *accum_ns,
                         unsigned long long *count, unsigned long long *raw_copy);

// Whole outer iterations in one persistent one-CTA launch, for tiny steps (mini_step.cu)
bool mini_step_ok(int32_t n, int32_t ldy, int32_t s, int32_t b, bool any_fit);
int launch_mini_steps(cudaStream_t st, const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n, int32_t ldy,
                      const int32_t *idx, int64_t n_steps, int32_t s, int32_t b, float alpha, int loss, int exact_margin,
                      float *x, uint16_t *xbf, int32_t ldxb, int split, uint16_t *Y, float *yI, float *G, int32_t ldg, float *r,
                      float *z, float *u, int *err_flag);

// s = 1 with wide rows: all iterations of a call in one persistent launch of one column-split cluster (s1_cluster.cu)
bool s1_cluster_ok(int32_t n, int32_t ldy, int32_t b, int cluster_max);
int launch_s1_cluster(cudaStream_t st, const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n, int32_t ldy,
                      const int32_t *idx, int64_t n_steps, int32_t b, float alpha, int loss, int exact_margin, float *x,
                      uint16_t *xbf, int32_t ldxb, int split, uint16_t *Y, float *yI, float *r, float *z, float *u, int *err_flag);

// P > 1 (partition.cu): the payload [r; strict block-lower G] of Alg. 1 line 5, packed / unpacked / summed over ranks
int64_t payload_count(int32_t s, int32_t b);
int launch_payload_pack(cudaStream_t st, const float *G, int32_t ldg, const float *r, int32_t s, int32_t b, float *payload,
                        int num_sms);
int launch_payload_unpack(cudaStream_t st, float *G, int32_t ldg, float *r, int32_t s, int32_t b, const float *payload,
                          int num_sms);
int launch_reduce_peers(cudaStream_t st, const float *const *peers_host, int32_t P, float *out, int64_t count, int num_sms);
int launch_reduce_unpack(cudaStream_t st, const float *const *peers_host, int32_t P, float *G, int32_t ldg, float *r, int32_t s,
                         int32_t b, int num_sms);

// tcgen05 Gram + margin (gram_tc.cu). r == nullptr: no margin (the pipelined schedule computes r in a kernel of its own).
// The plan owns the TMA tensor maps of the Y workspace and of the
// BF16 shadow (a [16 x ldxb] buffer: row 0 = x_bf, rows 1..15 zero). ksplit_opt <= 0: choose automatically.
// s = 1: there is no correction, u = l'(r, y_I) -- the Gram kernels' margin epilogue can apply l' itself.
struct S1Fuse {
    int loss;
    const float *yI;
    float *z, *u;
};
struct GramTcPlan;
GramTcPlan *gram_tc_plan_create(const uint16_t *Y, int32_t ldy, int32_t n, int32_t sb_rows_alloc,
                                const uint16_t *xbf, int32_t ldxb, char *err, int errlen);
void gram_tc_plan_destroy(GramTcPlan *p);
int launch_gram_tc(cudaStream_t st, GramTcPlan *plan, int32_t row_base, int32_t sb, int32_t b, float *G, int32_t ldg, float *r,
                   int full_lower, int ksplit_opt, int num_sms, char *err, int errlen);

// gather + Gram + margin in one kernel for narrow rows (n <= 64): gram_tc.cu
int launch_gram_narrow(cudaStream_t st, const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n,
                       const int32_t *idx, const StepParams *ind, int64_t idx_off, int32_t sb, int32_t b,
                       const uint16_t *xbf, int32_t ldxb, uint16_t *Y, int32_t ldy, float *yI, float *G, int32_t ldg,
                       float *r, int full_lower, int *err_flag, const S1Fuse *s1);

// cta_group::2 Gram + margin for large shapes (gram_pair.cu): 256 x 256 / 256 x 512 tiles on CTA pairs, work lists
// built on the host. gram_pair_prepare (outside stream capture) returns the estimated cycles, or -1.
struct GramPairPlan;
GramPairPlan *gram_pair_plan_create(const uint16_t *Y, int32_t ldy, int32_t n, int32_t rows_alloc, const uint16_t *xbf,
                                    int32_t ldxb, int num_sms);
void gram_pair_plan_destroy(GramPairPlan *p);
int64_t gram_pair_prepare(GramPairPlan *pl, int32_t sb, int32_t b, int full_lower, int bn, int ksplit_opt, int *bn_out, bool no_margin);
int launch_gram_pair(cudaStream_t st, GramPairPlan *pl, int32_t row_base, int32_t sb, int32_t b, float *G, int32_t ldg, float *r,
                     int full_lower, int bn, int ksplit_opt, char *err, int errlen);

}  // namespace casgd

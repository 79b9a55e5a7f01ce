// casgd_api.cu -- the C ABI of include/casgd.h: argument checks, workspace ownership, stage
// sequencing, CUDA-graph replay and the host-buffer entry point. No arithmetic of the method
// lives here; every step of the path runs in the kernels of this directory.
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <functional>
#include <map>
#include <new>
#include <tuple>
#include <vector>

#include "common.cuh"

using namespace casgd;

namespace casgd {
thread_local unsigned long long *g_stamp = nullptr;
thread_local bool g_plain_launch = false;
thread_local cudaEvent_t g_completion_event = nullptr;
}

namespace {

struct StageEvent {
    int stage;
    cudaEvent_t start, stop;
};

struct GraphKey {
    int32_t s, b;
    uint32_t eta_bits;
    int32_t len;
    bool operator<(const GraphKey &o) const
    {
        return std::tie(s, b, eta_bits, len) < std::tie(o.s, o.b, o.eta_bits, o.len);
    }
};

struct GraphEntry {
    cudaGraphExec_t exec;
    int64_t kernels;
    int last_buf;                       // Y stage its last step used (casgd_debug_export reads that one)
};

inline int64_t round_up(int64_t v, int64_t q) { return (v + q - 1) / q * q; }

}  // namespace

// Guard bands: every per-step workspace is allocated with kGuardBytes of a known pattern before and after it, and
// casgd_debug_export(CASGD_DBG_GUARDS) counts the guard bytes that changed -- an out-of-bounds write next to a workspace
// (a ragged tail, an off-by-one row) shows up there. (compute-sanitizer is closed on the pool this was developed on.)
#ifndef CASGD_GUARD_BYTES
#define CASGD_GUARD_BYTES 1024
#endif
constexpr size_t kGuardBytes = CASGD_GUARD_BYTES;
constexpr int kGuardPattern = 0xA5;
struct Guarded {
    unsigned char *base;                // start of the allocation
    size_t front;                       // bytes before the payload (its last kGuardBytes are the front guard)
    size_t bytes;                       // payload bytes
};

struct casgd_ctx {
    int device = 0;
    std::vector<Guarded> guarded;
    cudaStream_t stream = nullptr;
    cudaStream_t capture_stream = nullptr;
    cudaStream_t side_stream = nullptr;       // graph capture only: the branch that gathers the next step's rows
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    cudaStream_t gather_stream = nullptr;     // ... and the branch that gathers the rows of the step after next
    cudaEvent_t ev_gather[3] = {nullptr, nullptr, nullptr}, ev_gram[2] = {nullptr, nullptr}, ev_grad = nullptr, ev_rec_launch = nullptr;
    // dataset
    const uint16_t *A = nullptr;      // BF16 bits, row stride lda (borrowed or owned)
    uint16_t *A_owned = nullptr;
    int64_t lda = 0;
    const uint16_t *X_caller = nullptr;   // the caller's matrix when A is a repacked copy (casgd_loss streams narrow rows from it)
    int64_t ldx_caller = 0;
    const float *y = nullptr;
    int64_t m = 0;
    int32_t n = 0;
    int loss = 0;
    float *A32 = nullptr;             // lazy FP32 widening for the baseline
    // per-step workspaces, sized for rows_alloc rows
    int32_t rows_alloc = 0;
    int32_t ldy = 0, ldg = 0;
    uint16_t *Y = nullptr;            // THREE stages of rows_alloc rows (and of y_I), two of G: in the pipelined graphs step h
                                      // uses Y stage h % 3 and G stage h & 1 (a stage index below is y | g << 2)
    float *yI = nullptr, *G = nullptr, *r = nullptr, *z = nullptr, *u = nullptr;     // G, y_I: two stages as well
    float *r_scratch = nullptr;       // pipelined schedule: where the Gram kernels' fused margin (of a stale x) goes
    uint16_t *xbf = nullptr;          // BF16 shadow of x: [16 x ldxb], row 0 = bf16(x), the rest zero
    int32_t ldxb = 0;
    const float *shadow_of = nullptr;
    bool shadow_valid = false;
    GradWorkspace gws{};
    RecWorkspace rws{};
    StepParams *ind = nullptr;
    bool shadow_fresh = false;        // the shadow was built by the call in progress (host entry point)
    const int32_t *ind_idx = nullptr; // what the StepParams block on the device currently holds
    float *ind_x = nullptr;
    int *err_flag = nullptr;          // device alias of err_flag_host
    int *err_flag_host = nullptr;     // pinned, mapped
    double *loss_partials = nullptr, *loss_result = nullptr;
    double *loss_result_host = nullptr;   // pinned
    int32_t loss_max_blocks = 0;
    // host-buffer entry point staging
    int32_t *idx_stage = nullptr;
    int64_t idx_stage_cap = 0;
    float *x_stage = nullptr;
    float *x_snap = nullptr;          // CASGD_OPT_SNAPSHOT: x as it entered the last step of the last graph
    // last step, for debug export
    int32_t last_s = 0, last_b = 0, last_buf = 0;
    // options
    unsigned long long *stamps = nullptr;     // CASGD_OPT_STAMPS: [kStampSteps * 8][2] slots, accum_ns[8], count[8], raw copy of the slots
    int cur_slot_step = 0;                    // step index (inside the graph being captured) the next stage stamps into
    int64_t opt_stamps = 0;
    int64_t opt_gram_impl = 0, opt_full_lower = 0, opt_profile = 0, opt_no_graph = 0, opt_ksplit = 0, opt_rec_impl = 0, opt_loss_impl = 0, opt_no_fuse = 0, opt_overlap = 2, opt_chain_sms = 0, opt_split = 0, opt_mini = 1, opt_snapshot = 0;
    GramTcPlan *tc_plan = nullptr;
    GramPairPlan *pair_plans[2] = {nullptr, nullptr};   // work lists for all SMs [0] and for the pipelined schedule's share [1]
    GramPairPlan *first_gram_plan = nullptr;            // pipelined graphs: the whole-chip list of a graph's first Gram (or null)
    int pair_plan_sms[2] = {0, 0};
    GramPairPlan *pair_plan = nullptr;                  // the one of the schedule being enqueued
    int num_sms = 0;
    int gram_sms = 0, chain_sms = 0;  // SM budgets of the two branches for the shape being enqueued (both num_sms unless pipelined)
    int cur_gram = 0, cur_bn = 0;     // Gram kernel of the shape being enqueued: 1 = CUDA cores, 2 = 128x128 tiles, 3 = CTA pairs
    std::map<GraphKey, GraphEntry> graphs;
    std::vector<StageEvent> events;
    double stage_ms[CASGD_NUM_STAGES] = {};
    int64_t stage_launches[CASGD_NUM_STAGES] = {};
    int64_t launches = 0;
    char err[512] = "";
};

namespace {

constexpr int kRecReplicas = 8;
constexpr int kStampSteps = 64;                         // the longest graph
constexpr int kSlotStages = 8;                          // stamp slots per step (stages 0 .. 4 are stamped)
constexpr int kStampSlots = kStampSteps * kSlotStages;
constexpr int kStampAcc = 2 * kStampSlots;              // accum_ns[8], then count[8], then the raw copy of the last collect
constexpr int kStampRaw = kStampAcc + 16;
constexpr int kStampWords = kStampRaw + 2 * kStampSlots;
const unsigned kEpochInit[2] = {1u, 0u};                // {epoch, done}

int fail(casgd_ctx *c, int code, const char *fmt, ...)
{
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof c->err, fmt, ap);
        va_end(ap);
    }
    return code;
}

#define CK(call)                                                                                       \
    do {                                                                                               \
        cudaError_t e_ = (call);                                                                       \
        if (e_ != cudaSuccess)                                                                         \
            return fail(c, e_ == cudaErrorMemoryAllocation ? CASGD_ENOMEM : CASGD_ECUDA, "%s: %s", #call, \
                        cudaGetErrorString(e_));                                                       \
    } while (0)

void drop_graphs(casgd_ctx *c)
{
    for (auto &kv : c->graphs) cudaGraphExecDestroy(kv.second.exec);
    c->graphs.clear();
}

// The payload of a large workspace keeps the 2 MB alignment cudaMalloc gave the allocation: with Y, G a mere 1 KB off it
// the pair Gram kernel ran 15 % slower beside the chain (82.7 against 72.1 us, measured) -- so the front pad is 2 MB there.
template <typename T>
cudaError_t alloc_guarded(casgd_ctx *c, T **out, size_t bytes)
{
    unsigned char *base = nullptr;
    const size_t padded = (bytes + 255) & ~(size_t)255;
    const size_t front = bytes >= (1u << 20) ? (size_t)2 << 20 : kGuardBytes;
    cudaError_t e = cudaMalloc(&base, front + padded + kGuardBytes);
    if (e != cudaSuccess) return e;
    if (kGuardBytes) {
        cudaMemset(base + front - kGuardBytes, kGuardPattern, kGuardBytes);
        cudaMemset(base + front + bytes, kGuardPattern, padded - bytes + kGuardBytes);
    }
    c->guarded.push_back(Guarded{base, front, bytes});
    *out = reinterpret_cast<T *>(base + front);
    return cudaSuccess;
}

void free_guarded(casgd_ctx *c)
{
    for (const Guarded &g : c->guarded) cudaFree(g.base);
    c->guarded.clear();
}

// guard bytes that no longer hold the pattern
int64_t count_guard_damage(casgd_ctx *c)
{
    int64_t bad = 0;
    std::vector<unsigned char> h;
    for (const Guarded &g : c->guarded) {
        const size_t padded = (g.bytes + 255) & ~(size_t)255;
        const size_t tail = padded - g.bytes + kGuardBytes;
        h.resize(kGuardBytes + tail);
        if (cudaMemcpy(h.data(), g.base + g.front - kGuardBytes, kGuardBytes, cudaMemcpyDeviceToHost) != cudaSuccess ||
            cudaMemcpy(h.data() + kGuardBytes, g.base + g.front + g.bytes, tail, cudaMemcpyDeviceToHost) != cudaSuccess)
            return -1;
        for (unsigned char v : h) bad += v != kGuardPattern;
    }
    return bad;
}

void free_step_workspace(casgd_ctx *c)
{
    drop_graphs(c);
    if (c->tc_plan) { gram_tc_plan_destroy(c->tc_plan); c->tc_plan = nullptr; }
    for (GramPairPlan *&pl : c->pair_plans) { if (pl) gram_pair_plan_destroy(pl); pl = nullptr; }
    c->pair_plan = nullptr;
    free_guarded(c);
    c->Y = nullptr; c->yI = c->G = c->r = c->z = c->u = c->r_scratch = nullptr;
    c->rows_alloc = 0;
}

int ensure_workspace(casgd_ctx *c, int32_t sb)
{
    if (sb <= c->rows_alloc) return CASGD_OK;
    CK(cudaStreamSynchronize(c->stream));
    free_step_workspace(c);
    const int32_t rows = (int32_t)round_up(sb, 2 * kTile);   // whole 256-row pair tiles: a tile never straddles the two stages
    c->ldg = rows;
    CK(alloc_guarded(c, &c->Y, sizeof(uint16_t) * (size_t)3 * rows * c->ldy));
    CK(alloc_guarded(c, &c->yI, sizeof(float) * 3 * rows));
    CK(alloc_guarded(c, &c->G, sizeof(float) * (size_t)2 * rows * rows));
    CK(alloc_guarded(c, &c->r, sizeof(float) * rows));
    CK(alloc_guarded(c, &c->r_scratch, sizeof(float) * rows));
    CK(alloc_guarded(c, &c->z, sizeof(float) * rows));
    CK(alloc_guarded(c, &c->u, sizeof(float) * rows));
    CK(cudaMemsetAsync(c->Y, 0, sizeof(uint16_t) * (size_t)3 * rows * c->ldy, c->stream));
    CK(cudaMemsetAsync(c->G, 0, sizeof(float) * (size_t)2 * rows * rows, c->stream));
    CK(cudaMemsetAsync(c->r_scratch, 0, sizeof(float) * rows, c->stream));
    CK(cudaMemsetAsync(c->yI, 0, sizeof(float) * 3 * rows, c->stream));
    CK(cudaMemsetAsync(c->r, 0, sizeof(float) * rows, c->stream));
    CK(cudaMemsetAsync(c->z, 0, sizeof(float) * rows, c->stream));
    CK(cudaMemsetAsync(c->u, 0, sizeof(float) * rows, c->stream));
    c->rows_alloc = rows;
    return CASGD_OK;
}

int check_step_args(casgd_ctx *c, const void *idx, const void *x, int64_t n_steps, int32_t s, int32_t b, float eta)
{
    if (!c) return CASGD_EINVAL;
    if (!idx || !x) return fail(c, CASGD_EINVAL, "idx and x must not be null");
    if (n_steps < 0) return fail(c, CASGD_EINVAL, "n_steps = %lld < 0", (long long)n_steps);
    if (s < 1 || b < 1) return fail(c, CASGD_EINVAL, "s = %d and b = %d must be >= 1", s, b);
    if ((int64_t)s * b > CASGD_MAX_SB) return fail(c, CASGD_EINVAL, "s*b = %lld exceeds CASGD_MAX_SB = %d", (long long)s * b, CASGD_MAX_SB);
    if (!(eta == eta)) return fail(c, CASGD_EINVAL, "eta is NaN");
    return CASGD_OK;
}

struct StageTimer {
    casgd_ctx *c;
    int stage;
    StageEvent ev{};
    bool on;
    StageTimer(casgd_ctx *c_, int stage_) : c(c_), stage(stage_), on(c_->opt_profile != 0)
    {
        g_stamp = (c->opt_stamps && c->stamps && stage <= CASGD_STAGE_MARGIN) ? c->stamps + 2 * (c->cur_slot_step * kSlotStages + stage) : nullptr;
        if (!on) return;
        ev.stage = stage;
        cudaEventCreate(&ev.start);
        cudaEventCreate(&ev.stop);
        cudaEventRecord(ev.start, c->stream);
    }
    void done(int launches)
    {
        g_stamp = nullptr;
        c->launches += launches;
        if (!on) return;
        cudaEventRecord(ev.stop, c->stream);
        c->events.push_back(ev);
        c->stage_launches[stage] += launches;
    }
};

// Where a step finds its rows. `buf`: which of the two Y / y_I / G stages it uses; `gathered`: an earlier step's side branch
// has already gathered them; `next_idx_off` >= 0: this step gathers the NEXT step's rows (Alg. 1 line 2 of iteration t + 1
// depends on no result of iteration t) into the other stage on c->side_stream, beside its own recurrence and update.
struct StepIo {
    int buf = 0;
    bool gathered = false;
    int64_t next_idx_off = -1;
};

inline bool step_is_s1(const casgd_ctx *c, int32_t s)
{
    // s = 1: no Gram, no correction, u = l'(r, y_I): one kernel computes the margin and applies l' (the fused
    // gather + Gram kernel's epilogue for n <= 64, a warp-per-row kernel otherwise); a forced Gram kernel still runs
    return s == 1 && !c->opt_no_fuse && (c->cur_gram == 4 || c->opt_gram_impl == 0);
}
// pipelined schedule: not at s = 1 (no Gram), and not with the recurrence kernels that want the whole chip or trigger
// their dependents early (the grid-wide cooperative kernel, the plain-load cluster kernel)
constexpr int64_t kClusterFromBytes = 4096;            // s = 1: steps beyond this go to s1_cluster.cu first (measured)
inline bool pipelined_mode(const casgd_ctx *c, int32_t s, int32_t b)
{
    if (c->opt_overlap != 2 || s == 1 || c->num_sms < 64) return false;
    const bool fused = !c->opt_no_fuse && recurrence_fuses_update(s, b, c->ldg, c->ldy, c->rws, (int)c->opt_rec_impl);
    const int k = recurrence_kernel_choice(s, b, c->ldg, c->rws, (int)c->opt_rec_impl, fused);
    return k == 1 || k == 4 || k == 5;
}

// ---- the stages of one outer iteration (Alg. 1 lines 2-17), each on the stream it is given ----

int stage_gather(casgd_ctx *c, cudaStream_t st, const int32_t *idx, const StepParams *ind, int64_t idx_off, int32_t sb, int buf,
                 int sms, int64_t *kernels)
{
    StageTimer t(c, CASGD_STAGE_GATHER);
    const int yb = buf & 3;
    const int k = launch_gather(st, c->A, c->lda, c->y, c->m, c->n, idx, ind, idx_off, sb, c->Y + (size_t)yb * c->rows_alloc * c->ldy,
                                c->ldy, c->yI + (size_t)yb * c->rows_alloc, c->err_flag, sms);
    t.done(k); *kernels += k;
    return CASGD_OK;
}

// G (and r, into `r_out`) of the rows in stage `buf`; the narrow kernel gathers them itself
int stage_gram(casgd_ctx *c, cudaStream_t st, const int32_t *idx, const StepParams *ind, int64_t idx_off, int32_t s, int32_t b,
               int buf, float *r_out, int64_t *kernels)
{
    const int32_t sb = s * b;
    const int yb = buf & 3, gb = buf >> 2;
    uint16_t *Y = c->Y + (size_t)yb * c->rows_alloc * c->ldy;
    float *yI = c->yI + (size_t)yb * c->rows_alloc;
    float *G = c->G + (size_t)gb * c->rows_alloc * c->rows_alloc;
    const int32_t row_base = yb * c->rows_alloc;
    const S1Fuse s1f{c->loss, yI, c->z, c->u};
    int k;
    StageTimer t(c, CASGD_STAGE_GRAM);
    // r_out == nullptr: no margin wanted (pipelined schedule). The tcgen05 tile kernels then leave the x_bf rows out;
    // the narrow and CUDA-core kernels write theirs (of a stale x) to a scratch vector
    if (!r_out && (c->cur_gram == 4 || c->cur_gram == 1)) r_out = c->r_scratch;
    if (c->cur_gram == 4) {
        k = launch_gram_narrow(st, c->A, c->lda, c->y, c->m, c->n, idx, ind, idx_off, sb, b, c->xbf, c->ldxb, Y, c->ldy,
                               yI, G, c->ldg, r_out, (int)c->opt_full_lower, c->err_flag, step_is_s1(c, s) ? &s1f : nullptr);
        if (k < 0) return fail(c, CASGD_ECUDA, "gram_narrow launch: %s", cudaGetErrorString(cudaGetLastError()));
    } else if (c->cur_gram == 1) {
        k = launch_gram_simt(st, Y, c->ldy, c->n, sb, b, c->xbf, c->opt_split ? c->ldxb : 0, G, c->ldg, r_out, (int)c->opt_full_lower);
    } else if (c->cur_gram == 3) {
        k = launch_gram_pair(st, c->pair_plan, row_base, sb, b, G, c->ldg, r_out, (int)c->opt_full_lower, c->cur_bn,
                             (int)c->opt_ksplit, c->err, sizeof c->err);
        if (k < 0) return CASGD_ECUDA;
    } else {
        if (!c->tc_plan) {
            c->tc_plan = gram_tc_plan_create(c->Y, c->ldy, c->n, 3 * c->rows_alloc, c->xbf, c->ldxb, c->err, sizeof c->err);
            if (!c->tc_plan) return CASGD_ECUDA;
        }
        k = launch_gram_tc(st, c->tc_plan, row_base, sb, b, G, c->ldg, r_out, (int)c->opt_full_lower, (int)c->opt_ksplit, c->gram_sms, c->err, sizeof c->err);
        if (k < 0) return CASGD_ECUDA;
    }
    t.done(k); *kernels += k;
    return CASGD_OK;
}

int stage_margin(casgd_ctx *c, cudaStream_t st, const float *x, const StepParams *ind, int32_t sb, int buf, int64_t *kernels)
{
    StageTimer t(c, CASGD_STAGE_MARGIN);
    const int k = launch_margin(st, c->Y + (size_t)(buf & 3) * c->rows_alloc * c->ldy, c->ldy, c->n, sb, c->xbf, x, ind, c->opt_split != 0,
                                c->r, c->chain_sms);
    t.done(k); *kernels += k;
    return CASGD_OK;
}

// recurrence and update of the rows in stage `buf`
int stage_chain(casgd_ctx *c, cudaStream_t st, float *x, const StepParams *ind, int32_t s, int32_t b, float alpha, int buf,
                bool late_trigger, const std::function<void()> &after_recurrence, int64_t *kernels, bool force_recurrence = false,
                bool fuse_margin = false)
{
    const int32_t sb = s * b;
    uint16_t *Y = c->Y + (size_t)(buf & 3) * c->rows_alloc * c->ldy;
    float *yI = c->yI + (size_t)(buf & 3) * c->rows_alloc;
    float *G = c->G + (size_t)(buf >> 2) * c->rows_alloc * c->rows_alloc;
    int k;
    const bool fused = !c->opt_no_fuse && recurrence_fuses_update(s, b, c->ldg, c->ldy, c->rws, (int)c->opt_rec_impl);
    if (!step_is_s1(c, s) || force_recurrence) {
        StageTimer t(c, CASGD_STAGE_RECURRENCE);
        const FusedUpdate fu{Y, c->ldy, c->n, x, ind, c->xbf, c->opt_split ? c->ldxb : 0, fuse_margin ? c->r : nullptr};
        // late trigger: keep the dependent GRADIENT kernel's CTAs from becoming resident (and waiting) on SMs the side
        // branch needs. With the update fused in, the dependent is the next recurrence (after its Gram, a full edge):
        // let it launch early -- its launch latency is then off the chain (1.5 us per step on the chain-bound shapes)
        c->rws.late_trigger = late_trigger && !fused;
        c->rws.g_protected = c->cur_gram == 3;
        k = launch_recurrence(st, G, c->ldg, c->r, yI, s, b, alpha, c->loss, c->z, c->u, c->rws,
                              (int)c->opt_rec_impl, fused ? &fu : nullptr);
        g_completion_event = nullptr;
        if (k < 0) return fail(c, CASGD_ECUDA, "recurrence launch: %s", cudaGetErrorString(cudaGetLastError()));
        t.done(k); *kernels += k;
    }
    if (after_recurrence) after_recurrence();
    if (!fused) {
        StageTimer t(c, CASGD_STAGE_GRADIENT);
        c->gws.num_sms = c->chain_sms;
        c->gws.split_ld = c->opt_split ? c->ldxb : 0;
        k = launch_gradient_bf16(st, Y, c->ldy, c->n, sb, c->u, alpha, x, ind, c->xbf, c->gws);
        t.done(k); *kernels += k;
    }
    return CASGD_OK;
}

// Enqueue one outer iteration (Alg. 1 lines 2-17) on one stream (plus, with io.next_idx_off, the next step's gather on the
// side branch). `ind` non-null: graph-replay addressing.
int enqueue_step(casgd_ctx *c, cudaStream_t st, const int32_t *idx, const StepParams *ind, int64_t idx_off, float *x,
                 int32_t s, int32_t b, float eta, int64_t *kernels, const StepIo &io = StepIo{})
{
    const int32_t sb = s * b;
    const float alpha = eta / (float)b;
    int rc;
    c->last_buf = io.buf;
    const bool s1 = step_is_s1(c, s);
    if (s1 && c->cur_gram != 4) {
        // wide rows: gather + margin + l' in one warp-per-row kernel (there is no Gram at s = 1)
        StageTimer t(c, CASGD_STAGE_GRAM);
        const int k = launch_margin_s1(st, c->A, c->lda, c->y, c->m, c->n, idx, ind, idx_off, b, c->loss, c->xbf, c->opt_split ? c->ldxb : 0,
                                       c->Y + (size_t)(io.buf & 3) * c->rows_alloc * c->ldy, c->ldy, c->yI + (size_t)(io.buf & 3) * c->rows_alloc,
                                       c->r, c->z, c->u, c->err_flag);
        t.done(k); *kernels += k;
    } else {
        if (c->cur_gram != 4 && !io.gathered && (rc = stage_gather(c, st, idx, ind, idx_off, sb, io.buf, c->gram_sms, kernels))) return rc;
        if ((rc = stage_gram(c, st, idx, ind, idx_off, s, b, io.buf, c->r, kernels))) return rc;
    }
    const bool side = io.next_idx_off >= 0;
    std::function<void()> none;
    if (side) {
        // the next step's rows, on the side branch of the graph being captured
        cudaEventRecord(c->ev_fork, st);
        cudaStreamWaitEvent(c->side_stream, c->ev_fork, 0);
        const int saved_step = c->cur_slot_step;
        c->cur_slot_step = saved_step + 1;              // (stamps: the gather belongs to the next step)
        // the recurrence cluster holds up to 16 SMs: a gather sized for all SMs would leave 16 CTAs waiting for it to
        // finish (measured: 42 us instead of 12)
        rc = stage_gather(c, c->side_stream, idx, ind, io.next_idx_off, sb, (io.buf & 3) ^ 1, c->num_sms > 32 ? c->num_sms - 16 : c->num_sms, kernels);
        c->cur_slot_step = saved_step;
        if (rc) return rc;
        cudaEventRecord(c->ev_join, c->side_stream);
    }
    if ((rc = stage_chain(c, st, x, ind, s, b, alpha, io.buf, side, none, kernels))) return rc;
    if (side) cudaStreamWaitEvent(st, c->ev_join, 0);   // the next Gram needs the side branch's rows
    return CASGD_OK;
}

// CASGD_OPT_OVERLAP = 2: `len` outer iterations as a three-branch graph. G(t+1) = Y(t+1) Y(t+1)^T and Y(t+2) = A[I(t+2), :]
// need nothing iteration t computes, so the Gram branch runs Gram(t+1) on gram_sms SMs and the gather branch gather(t+2)
// on the chain's spare SMs while the main branch runs margin(t) -> recurrence(t) -> update(t); only r(t+1) = Y(t+1)
// x_bf(t+1) has to wait for the update. Three Y / y_I stages (h % 3), two G stages (h & 1).
//   Gram branch:    Gram(h+1) after gather(h+1), once every CTA of recurrence(h) is running (launch-completion event: the
//                   cluster needs its 16 SMs of one GPC before the Gram's persistent CTAs fill the chip)
//   gather branch:  gather(h+2) once recurrence(h) is running (hence after update(h-1), the last reader of its stage)
//   main:           margin(h) after gather(h); recurrence(h) after Gram(h); update(h)
// Side-branch kernels are launched without programmatic serialisation and the recurrence triggers its dependents late:
// a kernel that becomes resident early only to wait would hold SMs the other branch needs.
int capture_pipelined(casgd_ctx *c, int32_t s, int32_t b, float eta, int32_t len, int64_t *kernels)
{
    cudaStream_t M = c->capture_stream, S = c->side_stream, T = c->gather_stream;
    const int32_t sb = s * b;
    const float alpha = eta / (float)b;
    const bool has_gather = c->cur_gram != 4;           // (narrow rows: the Gram kernel gathers them itself)
    int rc = CASGD_OK;
    auto stage_of = [](int h) { return (h % 3) | ((h & 1) << 2); };      // Y stage h % 3, G stage h & 1
    cudaEventRecord(c->ev_fork, M);
    cudaStreamWaitEvent(S, c->ev_fork, 0);
    cudaStreamWaitEvent(T, c->ev_fork, 0);
    // gather(h) on the gather branch. h < 2: up front, on the Gram's share of the SMs; later ones run beside recurrence(h-2),
    // on the chain's SMs the cluster leaves free (so the side branch is the Gram alone)
    auto gather_step = [&](int h, bool beside_recurrence) -> int {
        if (!has_gather) return CASGD_OK;
        c->cur_slot_step = h;
        g_plain_launch = true;
        if (beside_recurrence) cudaStreamWaitEvent(T, c->ev_rec_launch, 0);
        const int sms = beside_recurrence ? std::max(8, c->chain_sms - 16) : c->num_sms;     // (up front: nothing else runs)
        const int rc2 = stage_gather(c, T, nullptr, c->ind, (int64_t)h * sb, sb, stage_of(h), sms, kernels);
        cudaEventRecord(c->ev_gather[h % 3], T);
        g_plain_launch = false;
        return rc2;
    };
    auto gram_step = [&](int h, bool wait_rec_launch) -> int {
        c->cur_slot_step = h;
        g_plain_launch = true;
        if (has_gather) cudaStreamWaitEvent(S, c->ev_gather[h % 3], 0);
        if (wait_rec_launch) cudaStreamWaitEvent(S, c->ev_rec_launch, 0);
        GramPairPlan *const shared_plan = c->pair_plan;
        if (!wait_rec_launch && c->cur_gram == 3 && c->first_gram_plan) c->pair_plan = c->first_gram_plan;
        const int rc2 = stage_gram(c, S, nullptr, c->ind, (int64_t)h * sb, s, b, stage_of(h), nullptr, kernels);
        c->pair_plan = shared_plan;
        cudaEventRecord(c->ev_gram[h & 1], S);
        if (!has_gather) cudaEventRecord(c->ev_gather[h % 3], S);
        g_plain_launch = false;
        return rc2;
    };
    rc = gather_step(0, false);
    if (!rc && len > 1) rc = gather_step(1, false);
    if (!rc) rc = gram_step(0, false);
    for (int32_t h = 0; h < len && rc == CASGD_OK; ++h) {
        const int buf = stage_of(h);
        c->cur_slot_step = h;
        cudaStreamWaitEvent(M, c->ev_gather[h % 3], 0);
        if (c->opt_snapshot && h + 1 == len) *kernels += launch_snapshot(M, nullptr, c->ind, c->n, c->x_snap);
        // small Y (the shapes whose update the recurrence cluster does itself): the cluster computes its rows' margin too
        // -- while a CTA's share of Y is a few KB (measured: n = 18, s*b = 2048, 8 KB per CTA: 21.1 -> 20.6 us per step;
        // n = 512, 128 KB per CTA: 26.3 -> 27.4, the 16 SMs of the cluster are slower at it than a kernel on 32)
        const bool fuse_margin = !c->opt_no_fuse && recurrence_fuses_update(s, b, c->ldg, c->ldy, c->rws, (int)c->opt_rec_impl) &&
                                 (int64_t)sb * c->ldy * 2 <= (int64_t)16 * 1024 * std::max(1, c->rws.cluster);
        if (!fuse_margin && (rc = stage_margin(c, M, nullptr, c->ind, sb, buf, kernels))) break;
        cudaStreamWaitEvent(M, c->ev_gram[h & 1], 0);
        const bool more = h + 1 < len;
        if (more) g_completion_event = c->ev_rec_launch;
        int rc_side = CASGD_OK;
        std::function<void()> after = [&]() {
            // once every CTA of recurrence(h) is running: the Gram of h + 1 (Y stage (h+1) % 3 gathered earlier, G stage
            // (h+1) & 1 last read by recurrence(h-1)) and the gather of h + 2 (Y stage (h+2) % 3, last read by update(h-1))
            if (more) rc_side = gram_step(h + 1, true);
            if (!rc_side && h + 2 < len) rc_side = gather_step(h + 2, true);
            c->cur_slot_step = h;
        };
        rc = stage_chain(c, M, nullptr, c->ind, s, b, alpha, buf, true, after, kernels, false, fuse_margin);
        if (!rc) rc = rc_side;
    }
    cudaEventRecord(c->ev_join, T);                     // every branch rejoins the origin stream before the capture ends
    cudaStreamWaitEvent(M, c->ev_join, 0);
    cudaEventRecord(c->ev_join, S);
    cudaStreamWaitEvent(M, c->ev_join, 0);
    c->last_buf = stage_of(len - 1);
    c->cur_slot_step = 0;
    g_plain_launch = false;
    g_completion_event = nullptr;
    return rc;
}

// Pick the Gram kernel for this shape (outside stream capture: the pair kernel's work list is uploaded here).
// CASGD_OPT_GRAM_IMPL: 0 = by the cost model, 1 = CUDA cores, 2 = 128x128 tcgen05 tiles, 3 / 4 = CTA pairs with
// 256 / 512-column tiles.
int choose_gram(casgd_ctx *c, int32_t s, int32_t b, bool pipe)
{
    const int32_t sb = s * b;
    const int64_t opt = c->opt_gram_impl;
    // SM budgets of the two branches. In the pipelined graphs (`pipe`) the chain keeps chain_sms SMs (the recurrence
    // cluster's 16 and a few more for the margin and update streams) and gather and Gram are sized for the rest; single
    // steps (and the sequential schedules) give every kernel the whole chip.
    c->gram_sms = c->chain_sms = c->num_sms;
    c->first_gram_plan = nullptr;
    c->cur_gram = 2;                                    // (pipelined_mode asks step_is_s1, which looks at cur_gram)
    pipe = pipe && pipelined_mode(c, s, b);
    if (pipe) {
        // The chain's share, measured. With the pair Gram's six-stage ring the Gram branch (68 us on 52 pairs) is no longer
        // the critical path of the headline shape; margin -> recurrence -> update is, and its two streaming kernels scale
        // with SMs while 46 pairs still hold the work list in three waves (120 whole tiles + 16 N = 128 items): synth-linear
        // s = 32 at 44 / 48 / 52 / 56 / 60 SMs: 76.5 / 75.6 / 74.3 / 73.8 / 82.3 us per step. Steps of a few MB gain nothing
        // from more chain SMs (epsilon-shaped s = 64: 43.3 at 44, 43.7 at 56): 56 from 16 MB of rows per step on, else 44.
        const int chain_default = (int64_t)sb * c->ldy * 2 >= ((int64_t)16 << 20) ? 56 : 44;
        const int chain = c->opt_chain_sms > 0 ? (int)c->opt_chain_sms : chain_default;
        c->chain_sms = std::min(std::max(chain, 16), c->num_sms - 32) & ~1;
        c->gram_sms = c->num_sms - c->chain_sms;
    }
    c->cur_gram = opt == 1 ? 1 : 2;
    c->cur_bn = 0;
    // gather + Gram in one kernel: wins while the tiles fit in about half a wave (measured at n = 18, b = 64: sb = 1536
    // 20.7 against 21.8 us per step, sb = 2048 29.8 against 25.7 us)
    if ((opt == 5 || (opt == 0 && sb <= 1536)) && c->n <= 64) { c->cur_gram = 4; return CASGD_OK; }
    if (opt == 5) return fail(c, CASGD_EINVAL, "the fused gather + Gram kernel needs n <= 64");
    if (opt == 1 || opt == 2 || c->gram_sms < 2) return CASGD_OK;
    if (opt == 0 && (sb < 512 || c->n < 256)) return CASGD_OK;      // too little work for 256-row tiles
    GramPairPlan *&plan = c->pair_plans[pipe ? 1 : 0];
    if (plan && c->pair_plan_sms[pipe ? 1 : 0] != c->gram_sms) { gram_pair_plan_destroy(plan); plan = nullptr; }
    if (!plan) {
        c->pair_plan_sms[pipe ? 1 : 0] = c->gram_sms;
        plan = gram_pair_plan_create(c->Y, c->ldy, c->n, 3 * c->rows_alloc, c->xbf, c->ldxb, c->gram_sms);
        if (!plan) return fail(c, CASGD_ECUDA, "cuTensorMapEncodeTiled failed for the pair Gram kernel");
    }
    c->pair_plan = plan;
    int bn = 0;
    const int64_t span = gram_pair_prepare(c->pair_plan, sb, b, (int)c->opt_full_lower, opt == 3 ? 256 : opt == 4 ? 512 : 0,
                                           (int)c->opt_ksplit, &bn, pipe);
    if (span < 0) {
        if (opt >= 3) return fail(c, CASGD_EINVAL, "the pair Gram kernel cannot run s*b = %d (work list too long)", sb);
        return CASGD_OK;
    }
    if (opt == 0) {
        // 128x128 tiles: 32 KB per K block per SM at the L2 cap of ~42.6 B/cycle/SM = 770 cycles
        const int64_t T = (sb + kTile - 1) / kTile, kbt = (c->n + 63) / 64;
        int64_t tiles = 0;
        for (int64_t ti = 0; ti < T; ++ti)
            for (int64_t tj = 0; tj <= ti; ++tj) {
                const int64_t last_row = std::min<int64_t>(ti * kTile + kTile, sb) - 1;
                tiles += (ti == tj) || c->opt_full_lower || (last_row / b) > (tj * kTile / b);
            }
        int64_t ks = std::max<int64_t>(1, std::min<int64_t>(c->gram_sms / std::max<int64_t>(tiles, 1), kbt / 16));
        if (ks > 1 && kbt - kbt / ks < 24) ks = 1;
        const int64_t span_tc = (tiles * ks + c->gram_sms - 1) / c->gram_sms * ((kbt + ks - 1) / ks) * 770 + 2600 + (ks > 1 ? 12000 : 0);
        // + the pair kernel's fixed cost (cluster launch, two cluster barriers, an epilogue nothing overlaps): ~12k cycles,
        // measured on one-tile-per-pair shapes (n = 2000, sb = 2048: 23 us against 18.8 us for the 128-tile kernel)
        if ((span + 12000) * 10 > span_tc * 9) return CASGD_OK;     // not clearly better: stay with the simpler kernel
    }
    c->cur_gram = 3;
    c->cur_bn = bn;
    // The FIRST Gram of a pipelined graph has the chip to itself (the chain it will run beside does not exist yet): it gets
    // a whole-chip work list of the same tiles (no margin items), so that a graph's pipeline fills in 12 + 47 instead of
    // 14 + 70 us (a 20-step graph: ~1.3 us per step)
    c->first_gram_plan = nullptr;
    if (pipe) {
        GramPairPlan *&full = c->pair_plans[0];
        if (full && c->pair_plan_sms[0] != c->num_sms) { gram_pair_plan_destroy(full); full = nullptr; }
        if (!full) {
            c->pair_plan_sms[0] = c->num_sms;
            full = gram_pair_plan_create(c->Y, c->ldy, c->n, 3 * c->rows_alloc, c->xbf, c->ldxb, c->num_sms);
        }
        int bn_full = 0;
        if (full && gram_pair_prepare(full, sb, b, (int)c->opt_full_lower, bn, (int)c->opt_ksplit, &bn_full, true) >= 0 && bn_full == bn)
            c->first_gram_plan = full;
    }
    return CASGD_OK;
}

// The BF16 shadow is rebuilt from x at the start of EVERY casgd_outer_step(s) call (one n-element kernel per call, not
// per step): a pointer-keyed cache would be fooled by an allocator that hands a new iterate the address of a freed one.
// The device alias of a pinned, mapped host pointer (what torch's pin_memory() and cudaHostAlloc give), or null.
void *mapped_alias(const void *host_ptr)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, host_ptr) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return at.type == cudaMemoryTypeHost ? at.devicePointer : nullptr;
}

// after a stream synchronize: has a kernel met a row index outside [0, m)? (the flag is mapped pinned host memory)
int index_error_check(casgd_ctx *c)
{
    volatile int *flag = c->err_flag_host;
    if (*flag) {
        *flag = 0;
        return fail(c, CASGD_EINDEX, "a row index outside [0, %lld) was gathered", (long long)c->m);
    }
    return CASGD_OK;
}

int ensure_shadow(casgd_ctx *c, const float *x)
{
    StageTimer t(c, CASGD_STAGE_OTHER);
    int k = launch_shadow(c->stream, x, nullptr, c->n, c->xbf, c->ldxb, (int)c->opt_split);
    t.done(k);
    c->shadow_of = x;
    c->shadow_valid = true;
    return CASGD_OK;
}

int get_graph(casgd_ctx *c, int32_t s, int32_t b, float eta, int32_t len, GraphEntry *out)
{
    GraphKey key{s, b, 0u, len};
    memcpy(&key.eta_bits, &eta, sizeof eta);
    auto it = c->graphs.find(key);
    if (it != c->graphs.end()) { *out = it->second; return CASGD_OK; }
    cudaGraph_t graph = nullptr;
    {   // kernel choice, SM budgets and work lists of this graph's schedule (outside the capture: lists are uploaded)
        const int rc0 = choose_gram(c, s, b, len > 1);
        if (rc0) return rc0;
    }
    // captured on a stream of the library's own (the caller's may be the legacy default stream, which cannot
    // be captured); nothing runs during capture, and replays are launched on the caller's stream
    if (!c->capture_stream) CK(cudaStreamCreateWithFlags(&c->capture_stream, cudaStreamNonBlocking));
    CK(cudaStreamBeginCapture(c->capture_stream, cudaStreamCaptureModeThreadLocal));
    int64_t kernels = 0;
    int rc = CASGD_OK;
    const int64_t saved = c->launches;
    const bool pipelined = pipelined_mode(c, s, b) && len > 1;
    // mode 1: steps that have a gather kernel of their own gather the NEXT step's rows on a side branch (two Y stages)
    const bool overlap = c->opt_overlap == 1 && c->cur_gram != 4 && !step_is_s1(c, s) && len > 1;
    if ((overlap || pipelined) && !c->side_stream) {
        cudaStreamCreateWithFlags(&c->side_stream, cudaStreamNonBlocking);
        cudaStreamCreateWithFlags(&c->gather_stream, cudaStreamNonBlocking);
        for (cudaEvent_t *e : {&c->ev_fork, &c->ev_join, &c->ev_gather[0], &c->ev_gather[1], &c->ev_gather[2], &c->ev_gram[0], &c->ev_gram[1],
                               &c->ev_grad, &c->ev_rec_launch})
            cudaEventCreateWithFlags(e, cudaEventDisableTiming);
    }
    if (pipelined) {
        rc = capture_pipelined(c, s, b, eta, len, &kernels);
    } else {
        for (int32_t h = 0; h < len && rc == CASGD_OK; ++h) {
            c->cur_slot_step = h;
            StepIo io;
            if (overlap) {
                io.buf = (h & 1) | ((h & 1) << 2);
                io.gathered = h > 0;
                io.next_idx_off = h + 1 < len ? (int64_t)(h + 1) * s * b : -1;
            }
            if (c->opt_snapshot && h + 1 == len) kernels += launch_snapshot(c->capture_stream, nullptr, c->ind, c->n, c->x_snap);
            rc = enqueue_step(c, c->capture_stream, nullptr, c->ind, (int64_t)h * s * b, nullptr, s, b, eta, &kernels, io);
        }
    }
    c->cur_slot_step = 0;
    c->launches = saved;                      // capture launches nothing; replays are counted
    cudaError_t e = cudaStreamEndCapture(c->capture_stream, &graph);
    if (rc != CASGD_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
    if (e != cudaSuccess) return fail(c, CASGD_ECUDA, "cudaStreamEndCapture: %s", cudaGetErrorString(e));
    GraphEntry ge{nullptr, kernels, c->last_buf};
    e = cudaGraphInstantiate(&ge.exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) return fail(c, CASGD_ECUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(e));
    c->graphs[key] = ge;
    *out = ge;
    return CASGD_OK;
}

int collect_events(casgd_ctx *c)
{
    for (auto &ev : c->events) {
        float ms = 0.f;
        cudaError_t e = cudaEventElapsedTime(&ms, ev.start, ev.stop);
        if (e == cudaSuccess) c->stage_ms[ev.stage] += ms;
        cudaEventDestroy(ev.start);
        cudaEventDestroy(ev.stop);
    }
    c->events.clear();
    return CASGD_OK;
}

int run_steps(casgd_ctx *c, const int32_t *idx, int64_t n_steps, float *x, int32_t s, int32_t b, float eta,
              bool allow_graph, int64_t graph_from = 2)
{
    const int32_t sb = s * b;
    if (n_steps == 0) return CASGD_OK;
    int rc = ensure_workspace(c, sb);
    if (rc) return rc;
    // tiny steps: all n_steps iterations in ONE persistent one-CTA launch (mini_step.cu) -- unless a kernel was asked for
    if (c->opt_mini && !c->opt_gram_impl && !c->opt_rec_impl && !c->opt_no_fuse && !c->opt_full_lower && !c->opt_profile &&
        c->lda % 8 == 0 && mini_step_ok(c->n, c->ldy, s, b, c->opt_mini == 2) &&
        !(s == 1 && (c->opt_mini == 3 || (c->opt_mini == 1 && (int64_t)b * c->ldy * 2 > kClusterFromBytes)) &&
          s1_cluster_ok(c->n, c->ldy, b, c->rws.cluster))) {    // (s = 1 beyond a few KB of rows: the cluster, below)
        c->cur_slot_step = 0;
        StageTimer t(c, CASGD_STAGE_GRAM);
        const int k = launch_mini_steps(c->stream, c->A, c->lda, c->y, c->m, c->n, c->ldy, idx, n_steps, s, b, eta / (float)b, c->loss,
                                        (int)c->opt_split, x, c->xbf, c->ldxb, (int)c->opt_split, c->Y, c->yI, c->G, c->ldg, c->r,
                                        c->z, c->u, c->err_flag);
        if (k < 0) return fail(c, CASGD_ECUDA, "mini_step launch: %s", cudaGetErrorString(cudaGetLastError()));
        t.done(k);
        if (c->opt_stamps)
            launch_stamp_collect(c->stream, c->stamps, kSlotStages, c->stamps + kStampAcc, c->stamps + kStampAcc + 8, c->stamps + kStampRaw);
        c->last_s = s; c->last_b = b; c->last_buf = 0;
        c->shadow_of = x; c->shadow_valid = true;
        CK(cudaGetLastError());
        return CASGD_OK;
    }
    // s = 1 with rows of >= 128 bytes: likewise one persistent launch, of one cluster that splits the columns (s1_cluster.cu)
    if (s == 1 && c->opt_mini && !c->opt_gram_impl && !c->opt_rec_impl && !c->opt_no_fuse && !c->opt_profile && c->lda % 8 == 0 &&
        s1_cluster_ok(c->n, c->ldy, b, c->rws.cluster)) {
        c->cur_slot_step = 0;
        StageTimer t(c, CASGD_STAGE_GRAM);
        const int k = launch_s1_cluster(c->stream, c->A, c->lda, c->y, c->m, c->n, c->ldy, idx, n_steps, b, eta / (float)b, c->loss,
                                        (int)c->opt_split, x, c->xbf, c->ldxb, (int)c->opt_split, c->Y, c->yI, c->r, c->z, c->u,
                                        c->err_flag);
        if (k < 0) return fail(c, CASGD_ECUDA, "s1_cluster launch: %s", cudaGetErrorString(cudaGetLastError()));
        t.done(k);
        if (c->opt_stamps)
            launch_stamp_collect(c->stream, c->stamps, kSlotStages, c->stamps + kStampAcc, c->stamps + kStampAcc + 8, c->stamps + kStampRaw);
        c->last_s = s; c->last_b = b; c->last_buf = 0;
        c->shadow_of = x; c->shadow_valid = true;
        CK(cudaGetLastError());
        return CASGD_OK;
    }
    rc = choose_gram(c, s, b, false);
    if (rc) return rc;
    // (rebuilt on every call -- the caller may have changed x, or handed over another tensor at the same address --
    // unless the host entry point has just built it together with its copy of x)
    if (c->shadow_fresh && c->shadow_of == x) rc = CASGD_OK;
    else rc = ensure_shadow(c, x);
    c->shadow_fresh = false;
    if (rc) return rc;
    c->last_s = s;
    c->last_b = b;
    int64_t done = 0;
    if (allow_graph && !c->opt_profile && !c->opt_no_graph && n_steps >= graph_from) {
        // 64-step graphs, then the remainder as ONE graph of its own length (cached by length): a pipelined graph spends
        // ~60 us filling its pipeline (two gathers and a Gram before the first chain), so a call of 20 steps is one
        // 20-step graph rather than 8 + 8 and four single steps (synth-linear s = 32: 84.6 -> ~77 us per step)
        const int32_t lens[2] = {64, (int32_t)(n_steps % 64)};
        if (c->graphs.size() > 96) drop_graphs(c);          // (a caller that varies n_steps endlessly: start over)
        for (int li = 0; li < 2; ++li) {
            const int32_t len = lens[li];
            if (len < 1 || n_steps - done < len) continue;
            GraphEntry ge;
            rc = get_graph(c, s, b, eta, len, &ge);
            if (rc) return rc;
            while (n_steps - done >= len) {
                if (c->ind_idx != idx + done * sb || c->ind_x != x) {      // (the same buffers as last time: nothing to rewrite)
                    c->launches += launch_set_params(c->stream, c->ind, idx + done * sb, x);
                    c->ind_idx = idx + done * sb;
                    c->ind_x = x;
                }
                CK(cudaGraphLaunch(ge.exec, c->stream));
                c->launches += ge.kernels;
                c->last_buf = ge.last_buf;
                if (c->opt_stamps)
                    launch_stamp_collect(c->stream, c->stamps, len * kSlotStages, c->stamps + kStampAcc, c->stamps + kStampAcc + 8, c->stamps + kStampRaw);
                done += len;
            }
        }
    }
    if (done < n_steps && (rc = choose_gram(c, s, b, false))) return rc;      // single steps: every kernel on the whole chip
    for (; done < n_steps; ++done) {
        int64_t kernels = 0;
        rc = enqueue_step(c, c->stream, idx + done * sb, nullptr, 0, x, s, b, eta, &kernels);
        if (rc) return rc;
        if (c->opt_stamps)
            launch_stamp_collect(c->stream, c->stamps, kSlotStages, c->stamps + kStampAcc, c->stamps + kStampAcc + 8, c->stamps + kStampRaw);
    }
    CK(cudaGetLastError());
    return CASGD_OK;
}

}  // namespace

// ------------------------------------------------------------------------- C ABI ---

extern "C" {

const char *casgd_version(void) { return "casgd-b200 0.3 (sm_100a)"; }

int casgd_init(casgd_ctx **out, const uint16_t *X_bf16, int64_t ldx, const float *y, int64_t m, int32_t n, int loss,
               void *cuda_stream)
{
    if (!out) return CASGD_EINVAL;
    *out = nullptr;
    if (!X_bf16 || !y || m < 1 || n < 1 || ldx < n || loss < 0 || loss > 2) return CASGD_EINVAL;
    if (m >= (1ll << 31)) return CASGD_EINVAL;              // every index buffer of the ABI is int32
    casgd_ctx *c = new (std::nothrow) casgd_ctx;
    if (!c) return CASGD_ENOMEM;
    auto bail = [&](int code) { casgd_destroy(c); return code; };
    cudaDeviceProp prop;
    if (cudaGetDevice(&c->device) != cudaSuccess || cudaGetDeviceProperties(&prop, c->device) != cudaSuccess)
        return bail(CASGD_ECUDA);
    if (prop.major != 10) return bail(CASGD_EARCH);
    c->num_sms = prop.multiProcessorCount;
    // opt-in shared-memory sizes and cluster sizes are per-device function attributes: set them on this device
    if (gather_configure() != cudaSuccess || gradient_configure() != cudaSuccess || gram_tc_configure() != cudaSuccess ||
        gram_pair_configure() != cudaSuccess || loss_configure() != cudaSuccess || recurrence_configure() != cudaSuccess ||
        recurrence_stream_configure() != cudaSuccess || recurrence_chain_configure() != cudaSuccess || mini_step_configure() != cudaSuccess || s1_cluster_configure() != cudaSuccess)
        return bail(CASGD_ECUDA);
    c->stream = (cudaStream_t)cuda_stream;
    c->y = y; c->m = m; c->n = n; c->loss = loss;
    c->ldy = (int32_t)round_up(n, 8);

    auto ck = [&](cudaError_t e) { return e == cudaSuccess; };
    const bool in_place = (ldx % 8 == 0) && ((uintptr_t)X_bf16 % 16 == 0);
    if (in_place) {
        c->A = X_bf16;
        c->lda = ldx;
    } else {
        // narrow rows get a power-of-two stride so that no row straddles a 128-byte line
        int64_t lda = round_up(n, 8);
        if (lda < 64) { int64_t p = 8; while (p < lda) p <<= 1; lda = p; }
        if (!ck(cudaMalloc(&c->A_owned, sizeof(uint16_t) * (size_t)m * lda))) return bail(CASGD_ENOMEM);
        c->launches += launch_repack(c->stream, X_bf16, ldx, m, n, c->A_owned, lda, c->num_sms);
        if (!ck(cudaStreamSynchronize(c->stream))) return bail(CASGD_ECUDA);
        c->A = c->A_owned;
        c->lda = lda;
        c->X_caller = X_bf16;
        c->ldx_caller = ldx;
    }
    c->ldxb = (int32_t)round_up(n, 64);
    const size_t xbf_elems = (size_t)16 * c->ldxb;
    c->gws.ldp = c->ldy;
    c->gws.max_splits = 128;
    c->gws.num_sms = c->num_sms;
    c->loss_max_blocks = c->num_sms * 4;
    const int n_counters = 8192 + 1;              // gradient column tiles, plus casgd_loss's finished-CTA counter
    bool ok = ck(cudaMalloc(&c->xbf, sizeof(uint16_t) * xbf_elems)) &&
              ck(cudaMemsetAsync(c->xbf, 0, sizeof(uint16_t) * xbf_elems, c->stream)) &&
              ck(cudaMalloc(&c->gws.partial, sizeof(float) * (size_t)c->gws.max_splits * c->gws.ldp)) &&
              ck(cudaMalloc(&c->gws.counters, sizeof(unsigned) * n_counters)) &&
              ck(cudaMemsetAsync(c->gws.counters, 0, sizeof(unsigned) * n_counters, c->stream)) &&
              ck(cudaMalloc(&c->ind, sizeof(StepParams))) &&
              ck(cudaMalloc(&c->rws.utag, sizeof(unsigned long long) * CASGD_MAX_SB * kRecReplicas)) &&
              ck(cudaMemsetAsync(c->rws.utag, 0, sizeof(unsigned long long) * CASGD_MAX_SB * kRecReplicas, c->stream)) &&
              ck(cudaMalloc(&c->rws.epoch, 2 * sizeof(unsigned))) &&
              ck(cudaMemcpyAsync(c->rws.epoch, kEpochInit, 2 * sizeof(unsigned), cudaMemcpyHostToDevice, c->stream)) &&
              ck(cudaHostAlloc(&c->err_flag_host, sizeof(int), cudaHostAllocMapped)) &&
              ck((*c->err_flag_host = 0, cudaHostGetDevicePointer(&c->err_flag, c->err_flag_host, 0))) &&
              ck(cudaMalloc(&c->loss_partials, sizeof(double) * c->loss_max_blocks)) &&
              ck(cudaMalloc(&c->loss_result, sizeof(double))) &&
              ck(cudaMallocHost(&c->loss_result_host, sizeof(double))) &&
              ck(cudaMalloc(&c->x_stage, sizeof(float) * (size_t)n)) &&
              ck(cudaMalloc(&c->x_snap, sizeof(float) * (size_t)n)) &&
              ck(cudaMalloc(&c->stamps, sizeof(unsigned long long) * kStampWords)) &&
              ck(cudaMemsetAsync(c->stamps, 0, sizeof(unsigned long long) * kStampWords, c->stream));
    if (!ok) return bail(CASGD_ENOMEM);
    c->rws.done = c->rws.epoch + 1;
    c->rws.nrep = kRecReplicas;
    c->rws.max_ctas = recurrence_max_coresident_ctas(prop.multiProcessorCount);
    c->rws.cluster = recurrence_cluster_size();
    c->rws.grid_threshold_bytes = 64 * 1024;
    if (!ck(cudaStreamSynchronize(c->stream))) return bail(CASGD_ECUDA);   // kEpochInit is consumed
    *out = c;
    return CASGD_OK;
}

int casgd_outer_step(casgd_ctx *c, const int32_t *idx, float *x, int32_t s, int32_t b, float eta)
{
    int rc = check_step_args(c, idx, x, 1, s, b, eta);
    if (rc) return rc;
    return run_steps(c, idx, 1, x, s, b, eta, false);
}

int casgd_outer_steps(casgd_ctx *c, const int32_t *idx, int64_t n_steps, float *x, int32_t s, int32_t b, float eta)
{
    int rc = check_step_args(c, idx, x, n_steps, s, b, eta);
    if (rc) return rc;
    return run_steps(c, idx, n_steps, x, s, b, eta, true);
}

int casgd_outer_steps_host(casgd_ctx *c, const int32_t *idx_host, int64_t n_steps, float *x_host, int32_t s, int32_t b,
                           float eta)
{
    int rc = check_step_args(c, idx_host, x_host, n_steps, s, b, eta);
    if (rc) return rc;
    const int64_t count = n_steps * s * b;
    if (count > c->idx_stage_cap) {
        CK(cudaStreamSynchronize(c->stream));
        cudaFree(c->idx_stage);
        c->idx_stage = nullptr;
        c->idx_stage_cap = 0;
        CK(cudaMalloc(&c->idx_stage, sizeof(int32_t) * (size_t)count));
        c->idx_stage_cap = count;
    }
    // small steps in pinned (mapped) host memory: kernels read and write the host buffers directly
    const int32_t *idx_alias = nullptr;
    float *x_alias = nullptr;
    if (count * 4 <= (64 << 10) && (int64_t)c->n * 4 <= (256 << 10)) {
        idx_alias = static_cast<const int32_t *>(mapped_alias(idx_host));
        x_alias = static_cast<float *>(mapped_alias(x_host));
    }
    const bool zero_copy = idx_alias && x_alias;
    if (zero_copy) {
        c->launches += launch_stage_in(c->stream, idx_alias, count, c->idx_stage, x_alias, c->n, c->x_stage, c->xbf, c->ldxb,
                                       (int)c->opt_split);
        c->shadow_of = c->x_stage;
        c->shadow_valid = true;
        c->shadow_fresh = true;
    } else {
        if (count > 0) CK(cudaMemcpyAsync(c->idx_stage, idx_host, sizeof(int32_t) * (size_t)count, cudaMemcpyHostToDevice, c->stream));
        CK(cudaMemcpyAsync(c->x_stage, x_host, sizeof(float) * (size_t)c->n, cudaMemcpyHostToDevice, c->stream));
        c->shadow_valid = false;              // x_stage was overwritten from the host
    }
    // (a call of ONE step too replays a graph here: one launch instead of five on a stream the host then waits for)
    rc = run_steps(c, c->idx_stage, n_steps, c->x_stage, s, b, eta, true, 1);
    if (rc) return rc;
    if (zero_copy) c->launches += launch_stage_out(c->stream, c->x_stage, c->n, x_alias);
    else CK(cudaMemcpyAsync(x_host, c->x_stage, sizeof(float) * (size_t)c->n, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return index_error_check(c);
}

int casgd_outer_steps_sampled(casgd_ctx *c, int64_t n_steps, float *x, int32_t s, int32_t b, float eta, uint64_t seed,
                              uint64_t first_step)
{
    int dummy = 0;
    int rc = check_step_args(c, &dummy, x, n_steps, s, b, eta);
    if (rc) return rc;
    const int64_t count = n_steps * s * b;
    if (count > c->idx_stage_cap) {
        CK(cudaStreamSynchronize(c->stream));
        cudaFree(c->idx_stage);
        c->idx_stage = nullptr;
        c->idx_stage_cap = 0;
        CK(cudaMalloc(&c->idx_stage, sizeof(int32_t) * (size_t)count));
        c->idx_stage_cap = count;
    }
    if (count > 0) c->launches += launch_sample_indices(c->stream, c->idx_stage, n_steps, s * b, c->m, seed, first_step);
    return run_steps(c, c->idx_stage, n_steps, x, s, b, eta, true);
}

// ---- P > 1: the outer iteration in two halves around the sum over ranks (Alg. 1 line 5) ----

int64_t casgd_payload_count(int32_t s, int32_t b)
{
    if (s < 1 || b < 1 || (int64_t)s * b > CASGD_MAX_SB) return -1;
    return payload_count(s, b);
}

int casgd_payload_alloc(int64_t count, float **payload_dev)
{
    if (!payload_dev || count < 1) return CASGD_EINVAL;
    *payload_dev = nullptr;
    const cudaError_t e = cudaMalloc(payload_dev, sizeof(float) * (size_t)count);
    return e == cudaSuccess ? CASGD_OK : e == cudaErrorMemoryAllocation ? CASGD_ENOMEM : CASGD_ECUDA;
}

int casgd_payload_free(float *payload_dev) { return cudaFree(payload_dev) == cudaSuccess ? CASGD_OK : CASGD_ECUDA; }

int casgd_ipc_export(const float *payload_dev, void *handle_host)
{
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "CUDA IPC handles are 64 bytes");
    if (!payload_dev || !handle_host) return CASGD_EINVAL;
    cudaIpcMemHandle_t h;
    if (cudaIpcGetMemHandle(&h, const_cast<float *>(payload_dev)) != cudaSuccess) return CASGD_ECUDA;
    memcpy(handle_host, &h, sizeof h);
    return CASGD_OK;
}

int casgd_ipc_open(const void *handle_host, float **peer_payload_dev)
{
    if (!handle_host || !peer_payload_dev) return CASGD_EINVAL;
    cudaIpcMemHandle_t h;
    memcpy(&h, handle_host, sizeof h);
    void *p = nullptr;
    if (cudaIpcOpenMemHandle(&p, h, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) return CASGD_ECUDA;
    *peer_payload_dev = static_cast<float *>(p);
    return CASGD_OK;
}

int casgd_ipc_close(float *peer_payload_dev)
{
    return cudaIpcCloseMemHandle(peer_payload_dev) == cudaSuccess ? CASGD_OK : CASGD_ECUDA;
}

int casgd_step_local(casgd_ctx *c, const int32_t *idx, const float *x, int32_t s, int32_t b, float *payload_out)
{
    int rc = check_step_args(c, idx, x, 1, s, b, 0.f);
    if (rc) return rc;
    if (!payload_out || ((uintptr_t)payload_out & 15)) return fail(c, CASGD_EINVAL, "payload_out must be a 16-byte aligned device pointer");
    const int32_t sb = s * b;
    if ((rc = ensure_workspace(c, sb)) || (rc = choose_gram(c, s, b, false)) || (rc = ensure_shadow(c, x))) return rc;
    c->last_s = s; c->last_b = b; c->last_buf = 0;
    int64_t kernels = 0;
    const bool narrow = c->cur_gram == 4;
    const bool split_margin = false;
    if (!narrow && (rc = stage_gather(c, c->stream, idx, nullptr, 0, sb, 0, c->gram_sms, &kernels))) return rc;
    if ((narrow || s > 1) && (rc = stage_gram(c, c->stream, idx, nullptr, 0, s, b, 0, split_margin ? nullptr : c->r, &kernels))) return rc;
    if ((split_margin || (s == 1 && !narrow)) && (rc = stage_margin(c, c->stream, x, nullptr, sb, 0, &kernels))) return rc;
    c->launches += launch_payload_pack(c->stream, c->G, c->ldg, c->r, s, b, payload_out, c->num_sms);
    CK(cudaGetLastError());
    return CASGD_OK;
}

int casgd_reduce_peers(casgd_ctx *c, const float *const *peer_payloads_host, int32_t P, int32_t s, int32_t b)
{
    if (!c) return CASGD_EINVAL;
    if (!peer_payloads_host || s < 1 || b < 1 || s * b > c->rows_alloc || s != c->last_s || b != c->last_b)
        return fail(c, CASGD_EINVAL, "casgd_reduce_peers: (s, b) must be those of the casgd_step_local just run");
    const int k = launch_reduce_unpack(c->stream, peer_payloads_host, P, c->G, c->ldg, c->r, s, b, c->num_sms);
    if (k < 0) return fail(c, CASGD_EINVAL, "casgd_reduce_peers: P = %d must be in [1, 64] and every payload pointer non-null", P);
    c->launches += k;
    CK(cudaGetLastError());
    return CASGD_OK;
}

int casgd_step_finish(casgd_ctx *c, float *x, int32_t s, int32_t b, float eta, const float *payload_in)
{
    int dummy = 0;
    int rc = check_step_args(c, &dummy, x, 1, s, b, eta);
    if (rc) return rc;
    if (s != c->last_s || b != c->last_b || s * b > c->rows_alloc)
        return fail(c, CASGD_EINVAL, "casgd_step_finish: (s, b) must be those of the casgd_step_local just run");
    if (payload_in) c->launches += launch_payload_unpack(c->stream, c->G, c->ldg, c->r, s, b, payload_in, c->num_sms);
    int64_t kernels = 0;
    std::function<void()> none;
    rc = stage_chain(c, c->stream, x, nullptr, s, b, eta / (float)b, 0, false, none, &kernels, true);
    if (rc) return rc;
    CK(cudaGetLastError());
    return CASGD_OK;
}

int casgd_sgd_steps_fp32(casgd_ctx *c, const int32_t *idx, int64_t n_steps, float *x, int32_t b, float eta)
{
    int rc = check_step_args(c, idx, x, n_steps, 1, b, eta);
    if (rc) return rc;
    if (!c->A32) {
        CK(cudaMalloc(&c->A32, sizeof(float) * (size_t)c->m * c->lda));
        c->launches += launch_widen(c->stream, c->A, c->lda, c->m, c->n, c->A32, c->lda, c->num_sms);
    }
    rc = ensure_workspace(c, b);
    if (rc) return rc;
    c->shadow_valid = false;                  // x changes without the shadow following
    c->gws.num_sms = c->num_sms;
    const float alpha = eta / (float)b;
    for (int64_t h = 0; h < n_steps; ++h)
        c->launches += launch_sgd32_step(c->stream, c->A32, c->lda, c->y, c->m, c->n, idx + h * b, b, alpha, c->loss, x,
                                         c->u, c->z, c->err_flag, c->gws);
    CK(cudaGetLastError());
    return CASGD_OK;
}

int casgd_sgd_step_fp32(casgd_ctx *c, const int32_t *idx, float *x, int32_t b, float eta)
{
    return casgd_sgd_steps_fp32(c, idx, 1, x, b, eta);
}

int casgd_loss(casgd_ctx *c, const float *x, double *loss_host)
{
    if (!c) return CASGD_EINVAL;
    if (!x || !loss_host) return fail(c, CASGD_EINVAL, "x and loss_host must not be null");
    {
        StageTimer t(c, CASGD_STAGE_LOSS);
        t.done(launch_loss(c->stream, c->A, c->lda, c->X_caller, c->ldx_caller, c->y, c->m, c->n, c->loss, x,
                           c->loss_partials, c->loss_max_blocks, c->loss_result, c->gws.counters + 8192,
                           (int)c->opt_loss_impl, c->num_sms));
    }
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(c->loss_result_host, c->loss_result, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    *loss_host = *c->loss_result_host;
    return CASGD_OK;
}

int casgd_invalidate_shadow(casgd_ctx *c)
{
    if (!c) return CASGD_EINVAL;
    c->shadow_valid = false;
    return CASGD_OK;
}

int casgd_sync(casgd_ctx *c)
{
    if (!c) return CASGD_EINVAL;
    CK(cudaStreamSynchronize(c->stream));
    return index_error_check(c);
}

int casgd_debug_export(casgd_ctx *c, int what, void *dst_host, int64_t dst_bytes)
{
    if (!c) return CASGD_EINVAL;
    if (!dst_host) return fail(c, CASGD_EINVAL, "dst_host is null");
    const int64_t sb = (int64_t)c->last_s * c->last_b;
    if (sb == 0 && what != CASGD_DBG_XBF && what != CASGD_DBG_STAMPS && what != CASGD_DBG_GUARDS && what != CASGD_DBG_XSNAP) return fail(c, CASGD_EINVAL, "no outer step has run yet");
    CK(cudaStreamSynchronize(c->stream));
    auto need = [&](int64_t bytes) { return dst_bytes == bytes; };
    switch (what) {
    case CASGD_DBG_Y:
        if (!need(sb * c->n * 2)) break;
        CK(cudaMemcpy2D(dst_host, (size_t)c->n * 2, c->Y + (size_t)(c->last_buf & 3) * c->rows_alloc * c->ldy, (size_t)c->ldy * 2, (size_t)c->n * 2, (size_t)sb, cudaMemcpyDeviceToHost));
        return CASGD_OK;
    case CASGD_DBG_G:
        if (!need(sb * sb * 4)) break;
        CK(cudaMemcpy2D(dst_host, (size_t)sb * 4, c->G + (size_t)(c->last_buf >> 2) * c->rows_alloc * c->rows_alloc, (size_t)c->ldg * 4, (size_t)sb * 4, (size_t)sb, cudaMemcpyDeviceToHost));
        return CASGD_OK;
    case CASGD_DBG_YLAB: case CASGD_DBG_R: case CASGD_DBG_Z: case CASGD_DBG_U: {
        if (!need(sb * 4)) break;
        const float *src = what == CASGD_DBG_YLAB ? c->yI + (size_t)(c->last_buf & 3) * c->rows_alloc : what == CASGD_DBG_R ? c->r : what == CASGD_DBG_Z ? c->z : c->u;
        CK(cudaMemcpy(dst_host, src, (size_t)sb * 4, cudaMemcpyDeviceToHost));
        return CASGD_OK;
    }
    case CASGD_DBG_GUARDS: {
        if (!need(8)) break;
        const int64_t bad = count_guard_damage(c);
        if (bad < 0) return fail(c, CASGD_ECUDA, "reading the guard bands failed");
        *reinterpret_cast<int64_t *>(dst_host) = bad;
        return CASGD_OK;
    }
    case CASGD_DBG_XSNAP:
        if (!need((int64_t)c->n * 4)) break;
        CK(cudaMemcpy(dst_host, c->x_snap, (size_t)c->n * 4, cudaMemcpyDeviceToHost));
        return CASGD_OK;
    case CASGD_DBG_STAMPS:
        if (!need((int64_t)kStampSlots * 16)) break;
        CK(cudaMemcpy(dst_host, c->stamps + kStampRaw, (size_t)kStampSlots * 16, cudaMemcpyDeviceToHost));
        return CASGD_OK;
    case CASGD_DBG_XBF:
        if (!need((int64_t)c->n * 2)) break;
        CK(cudaMemcpy(dst_host, c->xbf, (size_t)c->n * 2, cudaMemcpyDeviceToHost));
        return CASGD_OK;
    default:
        return fail(c, CASGD_EINVAL, "unknown debug item %d", what);
    }
    return fail(c, CASGD_EINVAL, "dst_bytes = %lld does not match item %d of the last step (s = %d, b = %d, n = %d)",
                (long long)dst_bytes, what, c->last_s, c->last_b, c->n);
}

int casgd_set_option(casgd_ctx *c, int option, int64_t value)
{
    if (!c) return CASGD_EINVAL;
    switch (option) {
    case CASGD_OPT_GRAM_IMPL:
        if (value < 0 || value > 5) return fail(c, CASGD_EINVAL, "CASGD_OPT_GRAM_IMPL must be in [0, 5]");
        c->opt_gram_impl = value; break;
    case CASGD_OPT_GRAM_FULL_LOWER: c->opt_full_lower = value != 0; break;
    case CASGD_OPT_PROFILE:
        c->opt_profile = value != 0;
        break;
    case CASGD_OPT_NO_GRAPH: c->opt_no_graph = value != 0; break;
    case CASGD_OPT_GRAM_KSPLIT:
        if (value < 0 || value > 64) return fail(c, CASGD_EINVAL, "CASGD_OPT_GRAM_KSPLIT must be in [0, 64]");
        c->opt_ksplit = value; break;
    case CASGD_OPT_RECURRENCE_IMPL:
        if (value < 0 || value > 5) return fail(c, CASGD_EINVAL, "CASGD_OPT_RECURRENCE_IMPL must be in [0, 5]");
        c->opt_rec_impl = value; break;
    case CASGD_OPT_NO_FUSED_UPDATE: c->opt_no_fuse = value != 0; break;
    case CASGD_OPT_STAMPS:
        c->opt_stamps = value != 0;
        // arm every slot ({~0, 0}) and clear the totals: a collect pass over all slots, then zero the accumulators
        CK(cudaStreamSynchronize(c->stream));
        launch_stamp_collect(c->stream, c->stamps, kStampSlots, c->stamps + kStampAcc, c->stamps + kStampAcc + 8, c->stamps + kStampRaw);
        CK(cudaMemsetAsync(c->stamps + kStampAcc, 0, sizeof(unsigned long long) * 16, c->stream));
        break;
    case CASGD_OPT_OVERLAP:
        if (value < 0 || value > 2) return fail(c, CASGD_EINVAL, "CASGD_OPT_OVERLAP must be 0, 1 or 2");
        c->opt_overlap = value; break;
    case CASGD_OPT_MARGIN_SPLIT: c->opt_split = value != 0; break;
    case CASGD_OPT_MINI: c->opt_mini = value < 0 ? 0 : value > 3 ? 3 : value; break;
    case CASGD_OPT_SNAPSHOT: c->opt_snapshot = value != 0; break;
    case CASGD_OPT_CHAIN_SMS:
        if (value < 0 || value > 1024) return fail(c, CASGD_EINVAL, "CASGD_OPT_CHAIN_SMS must be in [0, 1024]");
        c->opt_chain_sms = value; break;
    case CASGD_OPT_LOSS_IMPL:
        if (value != 0 && value != 1) return fail(c, CASGD_EINVAL, "CASGD_OPT_LOSS_IMPL must be 0 or 1");
        c->opt_loss_impl = value; break;
    default: return fail(c, CASGD_EINVAL, "unknown option %d", option);
    }
    drop_graphs(c);
    return CASGD_OK;
}

int casgd_stage_times(casgd_ctx *c, double *ms_host, int64_t *launches_host, int reset)
{
    if (!c) return CASGD_EINVAL;
    CK(cudaStreamSynchronize(c->stream));
    collect_events(c);
    if (c->opt_stamps) {
        // in-graph stamps replace the event times of the four step stages
        unsigned long long acc[16];
        CK(cudaMemcpy(acc, c->stamps + kStampAcc, sizeof acc, cudaMemcpyDeviceToHost));
        for (int i = 0; i <= CASGD_STAGE_MARGIN; ++i) {
            if (ms_host) ms_host[i] = (double)acc[i] * 1e-6;
            if (launches_host) launches_host[i] = (int64_t)acc[8 + i];
        }
        for (int i = CASGD_STAGE_MARGIN + 1; i < CASGD_NUM_STAGES; ++i) {
            if (ms_host) ms_host[i] = c->stage_ms[i];
            if (launches_host) launches_host[i] = c->stage_launches[i];
            if (reset) { c->stage_ms[i] = 0.0; c->stage_launches[i] = 0; }
        }
        if (reset) CK(cudaMemset(c->stamps + kStampAcc, 0, sizeof(unsigned long long) * 16));
        return CASGD_OK;
    }
    for (int i = 0; i < CASGD_NUM_STAGES; ++i) {
        if (ms_host) ms_host[i] = c->stage_ms[i];
        if (launches_host) launches_host[i] = c->stage_launches[i];
        if (reset) { c->stage_ms[i] = 0.0; c->stage_launches[i] = 0; }
    }
    return CASGD_OK;
}

int64_t casgd_launch_count(const casgd_ctx *c) { return c ? c->launches : 0; }

const char *casgd_last_error(const casgd_ctx *c) { return c ? c->err : "null context"; }

void casgd_destroy(casgd_ctx *c)
{
    if (!c) return;
    cudaStreamSynchronize(c->stream);
    collect_events(c);
    free_step_workspace(c);
    if (c->capture_stream) cudaStreamDestroy(c->capture_stream);
    if (c->side_stream) cudaStreamDestroy(c->side_stream);
    if (c->gather_stream) cudaStreamDestroy(c->gather_stream);
    for (cudaEvent_t e : {c->ev_fork, c->ev_join, c->ev_gather[0], c->ev_gather[1], c->ev_gather[2], c->ev_gram[0], c->ev_gram[1], c->ev_grad, c->ev_rec_launch})
        if (e) cudaEventDestroy(e);
    cudaFree(c->A_owned); cudaFree(c->A32); cudaFree(c->xbf);
    cudaFree(c->gws.partial); cudaFree(c->gws.counters); cudaFree(c->ind);
    cudaFree(c->rws.utag); cudaFree(c->rws.epoch); cudaFree(c->stamps);
    cudaFree(c->loss_partials); cudaFree(c->loss_result); cudaFree(c->idx_stage); cudaFree(c->x_stage); cudaFree(c->x_snap);
    if (c->err_flag_host) cudaFreeHost(c->err_flag_host);
    if (c->loss_result_host) cudaFreeHost(c->loss_result_host);
    delete c;
}

}  // extern "C"

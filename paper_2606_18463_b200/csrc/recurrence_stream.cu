// recurrence_stream.cu -- the s-step inner residual correction, Alg. 1 lines 6-15:
//   for j = 0..s-1:  z_j = r_j - alpha * sum_{k<j} G_{jk} u_k ;  u_j = l'(z_j, y_{I_j})          (all FP32, L236)
// as ONE thread-block cluster whose critical path never waits for global memory.
//
// The chain has s-1 dependent hops; what a hop costs is (a) how fast u_k gets from the SMs that produce it to
// the SMs that need it and (b) whether the G values the next block needs are already on chip when it lands.
//   (a) u travels between the CTAs of the cluster with st.async + mbarrier::complete_tx (distributed shared
//       memory, ~0.1 us) -- every CTA holds all of u in its own shared memory and one mbarrier per block.
//   (b) every warp streams its own part of G from L2 into a private shared-memory ring with 16-byte cp.async
//       (LDGSTS: each lane copies, and later reads back, its own 16 bytes, so the ring needs no barrier --
//       cp.async.wait_group is the only synchronisation), kDepth 512-byte chunks ahead of use and independent
//       of the chain (measured: plain 16-byte loads from 16 warps reach ~80 B/cycle/SM, a single-thread
//       cp.async.bulk producer only 1-25).
// Rows: each block's rows are dealt to the CTAs in groups of 4 consecutive rows (group q -> CTA q mod C), so the
// four u values of a group leave as ONE 16-byte st.async per destination CTA (measured: a hop with 4-byte stores
// costs 850 cycles in a 16-CTA cluster, with 16-byte stores 540). Work of one CTA:
//   critical warps  three per owned group, taking every third step: the newest kWin = 2 chunks of the step's rows
//                   (the last one holds block j-1), the bulk partial, one 5-level shuffle reduction for the 4 rows,
//                   l', and the broadcast of u;
//   bulk warps      every other warp (12, or 10 when the CTA owns two groups), each taking WHOLE steps in turn: all
//                   older 128-column chunks of the step's rows -- blocks <= j-2, whose u landed a hop or more
//                   earlier, so a bulk warp runs ahead of the chain -- then one reduction and one hand-over per
//                   step through shared memory + an mbarrier. Their issue rate, not L2, bounded the late steps:
//                   hence running pointers, whole steps per warp and all four schedulers.
// The strict block-lower G is read exactly once (L180). Needs b % 4 == 0 and at most 2 groups per CTA (b <= 128
// with 16 CTAs). For small steps the same cluster then applies the outer update (Alg. 1 lines 16-17): see FusedGrad.
#include "common.cuh"
#include "rec_cluster.cuh"

namespace casgd {

namespace {

constexpr int kWarps = 16;
constexpr int kThreads = 32 * kWarps;
constexpr int kQuad = 4;                                // rows per row group: one 16-byte remote store carries their u
constexpr int kMaxQuadsPerCta = 2;                      // row groups of one block owned by one CTA (b <= 8 * C)
constexpr int kBulkWarps = 12;                          // bulk warps per CTA at most: every warp that is not critical (12 with one row group, 10 with two)
constexpr int kChunk = 128;                             // columns per chunk
constexpr uint32_t kUnitBytes = kQuad * kChunk * 4u;    // one unit: 4 rows x 128 columns of G = 2 KB
constexpr int kWin = 2;                                 // chunks of a step the critical warps take: the newest 256 columns
constexpr int kCritPer = 3;                             // critical warps per row group, taking every third step
constexpr int kDepth = 4;                               // bulk warp: units of its ring (3 in flight)
constexpr int kCritDepth = 3;                           // critical warp: steps in flight (kWin units each)
constexpr int kPartDepth = 40;                          // steps of partial sums kept (a bulk warp finishes step j only after u_{j-3} landed)

struct StreamLayout {                   // byte offsets into dynamic shared memory (base 128-byte aligned)
    uint32_t u, ubar, pbar, part, cring, bring, total;
};

// qmax = row groups of a block per CTA at most (1 or 2): the rings are sized for it, so that s*b = 16384 still fits
__host__ __device__ inline StreamLayout stream_layout(int s, int b, int qmax)
{
    StreamLayout L;
    uint32_t o = 0;
    L.u = o;      o += 4u * (uint32_t)(s * b);
    o = (o + 7u) & ~7u;
    L.ubar = o;   o += 8u * (uint32_t)s;
    L.pbar = o;   o += 8u * (uint32_t)s;
    o = (o + 15u) & ~15u;
    L.part = o;   o += 16u * (uint32_t)(kPartDepth * qmax);                             // [step % depth][quad][4 rows]
    o = (o + 127u) & ~127u;
    L.cring = o;  o += (uint32_t)(kCritPer * qmax * kCritDepth * kWin) * kUnitBytes;
    L.bring = o;  o += (uint32_t)((qmax == 1 ? 12 : 10) * kDepth) * kUnitBytes;         // one ring per bulk warp
    L.total = o;
    return L;
}

__device__ __forceinline__ int num_chunks(int j, int b) { return (j * b + kChunk - 1) / kChunk; }

#ifdef CASGD_REC_TRACE
__device__ long long g_rec_trace[8192];
#define REC_TRACE(i) do { if (crank == 0 && (warp & 3) == 0 && (warp >> 2) < kCritPer && lane == 0 && (i) < 8192) g_rec_trace[(i)] = clock64(); } while (0)
#define REC_TRACE_B(i) do { if (crank == 0 && warp == 2 && lane == 0 && (i) < 8192) g_rec_trace[(i)] = clock64(); } while (0)
#else
#define REC_TRACE_B(i) do { } while (0)
#define REC_TRACE(i) do { } while (0)
#endif

// Sum acc[i] (row i of the group) over the 32 lanes in five shuffle levels (six shuffles): afterwards lane l
// holds the total of row l >> 3.
__device__ __forceinline__ float quad_reduce(const float (&a)[kQuad], int lane)
{
    const bool h16 = lane & 16, h8 = lane & 8;
    float k0 = h16 ? a[2] : a[0], k1 = h16 ? a[3] : a[1];
    const float s0 = h16 ? a[0] : a[2], s1 = h16 ? a[1] : a[3];
    k0 += __shfl_xor_sync(0xffffffffu, s0, 16);
    k1 += __shfl_xor_sync(0xffffffffu, s1, 16);
    float k = h8 ? k1 : k0;
    const float sd = h8 ? k0 : k1;
    k += __shfl_xor_sync(0xffffffffu, sd, 8);
    k += __shfl_xor_sync(0xffffffffu, k, 4);
    k += __shfl_xor_sync(0xffffffffu, k, 2);
    k += __shfl_xor_sync(0xffffffffu, k, 1);
    return k;
}

template <int LOSS>
__global__ void __launch_bounds__(kThreads, 1)
recurrence_stream_kernel(const float *G, int32_t ldg, const float *r,
                         const float *yI, int32_t s, int32_t b, float alpha, float *z,
                         float *u, const FusedGrad fg, unsigned long long *stamp, int late_trigger)
{
    extern __shared__ __align__(128) unsigned char rs_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int C = (int)cluster_nctarank(), crank = (int)cluster_ctarank();
    // The dependent kernel's CTAs become resident (and wait) once every CTA here has triggered. Normally that is wanted
    // at once; with the next step's gather on a side branch it is not: the waiting CTAs would hold the SMs the gather
    // needs (measured: the gather took 42 us instead of 12), so the trigger then comes after the chain.
    if (!(late_trigger & 1)) pdl_trigger();
    REC_TRACE(0);
    const int qmax = (b / kQuad + C - 1) / C;           // row groups of a block per CTA at most
    const StreamLayout L = stream_layout(s, b, qmax);
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(rs_smem);
    const uint32_t us = base + L.u, ubar = base + L.ubar, pbar = base + L.pbar, part = base + L.part;

    // row groups (4 consecutive rows of a block) are dealt to the CTAs: group q -> CTA q mod C
    const int nquads = b / kQuad;
    const int qpc = crank < nquads ? (nquads - crank + C - 1) / C : 0;     // groups of each block owned here
    const int ndst = min(C, nquads);                                       // CTAs that own rows
    const int bshift = (b & (b - 1)) == 0 ? __ffs(b) - 1 : -1;             // b a power of two: column -> block by shift
    auto block_of = [&](int col) { return bshift >= 0 ? (col >> bshift) : col / b; };

    // G is read exactly once (L180). Where the pair Gram kernel wrote it with L2::evict_last (bit 1 of late_trigger), these
    // loads release the lines again (evict_first); elsewhere they keep the default priority (measured: the hint alone costs
    // poisson-synth s = 32 0.8 %)
    const unsigned long long pol_g = l2_policy((late_trigger & 2) != 0);
    const int nbulk = qmax == 1 ? 12 : 10;              // 16 warps - 3 critical warps per row group, rounded to a multiple of qmax
    for (int k = threadIdx.x; k < s; k += kThreads) {
        mbar_init(ubar + 8u * k, 1);
        mbar_expect_tx(ubar + 8u * k, 4u * (uint32_t)b);
        mbar_init(pbar + 8u * k, (uint32_t)max(qpc, 1));      // one bulk warp per owned row group reports per step
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    pdl_wait();                                         // G, r and y_I come from the Gram and gather kernels
    stamp_begin(stamp);
    if (fg.r_fused) {
        // Alg. 1 line 3 for the rows THIS CTA's critical warps own (row group q -> CTA q mod C, every block): the
        // pipelined schedule's stand-alone margin kernel folded in when Y is small (one launch and its gap less on the chain)
        fused_margin_rows(fg, s * qpc * kQuad, [&](int t) {
            const int j = t / (qpc * kQuad), rem = t - j * (qpc * kQuad);
            return j * b + kQuad * (crank + (rem >> 2) * C) + (rem & 3);
        }, warp, lane, kWarps);
        __threadfence_block();
        __syncthreads();                                // the critical warps below read r through ld_dep
    }

    // Warp w runs on scheduler w & 3. Critical warps: (group gamma, parity e) -> warp gamma + 4 e.
    const int wsched = warp & 3, wslot = warp >> 2;
    const bool is_critical = wslot < kCritPer && wsched < qpc;
    // bulk warps: the non-critical warps, on all four schedulers (the chain's instructions are few; what bounded the
    // late steps was the bulk warps' own issue rate, 8 warps on 2 schedulers: ~33 B/cycle/SM out of L2)
    const int ncrit_below = min(wslot, kCritPer) * qpc + (wslot < kCritPer ? min(wsched, qpc) : 0);
    const int brank = warp - ncrit_below;               // rank among the non-critical warps
    const bool is_bulk = qpc > 0 && !is_critical && brank < nbulk;
    const int li = lane >> 3;                           // the row of a group this lane finalises / reports

    if (is_critical) {
        // ===== critical warp: row group gamma (4 rows), steps j = e, e + kCritPer, ...; the newest kWin chunks =====
        // While this warp finishes step j (stores, prefetch) and sets up step j + kCritPer -- including the window's
        // older chunks, whose u is already there -- the group's next critical warp is waiting for u_j:
        // a hop is wake + one chunk's dot + reduce + l' + one 16-byte store per CTA.
        const int gamma = wsched, e = wslot;
        const int q0 = kQuad * (crank + gamma * C);                 // first row of the group inside a block
        const uint32_t ring = base + L.cring + (uint32_t)((gamma * kCritPer + e) * kCritDepth * kWin) * kUnitBytes + (uint32_t)lane * 16u;
        const float *gbase = G + (int64_t)q0 * ldg + lane * 4;
        // remote addresses are linear in the shared::cluster window: map the two bases once
        const uint32_t rem_us = mapa_u32(us, (uint32_t)(lane < ndst ? lane : 0));
        const uint32_t rem_ubar = mapa_u32(ubar, (uint32_t)(lane < ndst ? lane : 0));
        int pj = e > 0 ? e : kCritPer, pslot = 0;       // next step to prefetch (step 0 has no chunk)
        auto prefetch_step = [&]() {
            if (pj < s) {
                const int len = pj * b;
                const int nch = num_chunks(pj, b);
                const float *src = gbase + (int64_t)len * ldg;
#pragma unroll
                for (int w = 0; w < kWin; ++w) {
                    const int c = nch - kWin + w;
                    if (c >= 0 && c * kChunk + lane * 4 < len) {
#pragma unroll
                        for (int i = 0; i < kQuad; ++i)
                            cp_async16_hint(ring + (uint32_t)(pslot * kWin + w) * kUnitBytes + (uint32_t)i * (kChunk * 4u),
                                            src + (int64_t)i * ldg + c * kChunk, pol_g);
                    }
                }
                pj += kCritPer;
            }
            cp_async_commit();                          // always: wait_group counts groups, empty ones included
            pslot = (pslot + 1 == kCritDepth) ? 0 : pslot + 1;
        };
#pragma unroll 1
        for (int i = 0; i < kCritDepth - 1; ++i) prefetch_step();
        float rr = 0.f, yy = 0.f;
        if (e < s) { rr = ld_dep(r + e * b + q0 + li); yy = ld_dep(yI + e * b + q0 + li); }

        __syncthreads();
        cluster_sync_all();                             // nobody signals a barrier that is not initialised yet
        REC_TRACE(1);

        int slot = 0, ready = 0;                        // blocks 0 .. ready-1 of u are complete in u_s (this warp's view)
#pragma unroll 1
        for (int j = e; j < s; j += kCritPer) {
            const int row = j * b + q0;
            float rr_next = 0.f, yy_next = 0.f;
            if (j + kCritPer < s) {
                rr_next = ld_dep(r + row + kCritPer * b + li);
                yy_next = ld_dep(yI + row + kCritPer * b + li);
            }
            float acc[kQuad] = {0.f, 0.f, 0.f, 0.f};
            if (j > 0) {
                const int len = j * b;
                const int nch = num_chunks(j, b);
                cp_async_wait<kCritDepth - 2>();        // the oldest outstanding step (this one) has landed
                const uint32_t sbase = ring + (uint32_t)(slot * kWin) * kUnitBytes;
                slot = (slot + 1 == kCritDepth) ? 0 : slot + 1;
                // the newest chunk's G: in registers before the wait
                const int cl = nch - 1;
                const bool mine = cl * kChunk + lane * 4 < len;
                float4 gl[kQuad];
#pragma unroll
                for (int i = 0; i < kQuad; ++i) {
                    gl[i] = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (mine) gl[i] = lds_f4(sbase + (uint32_t)(kWin - 1) * kUnitBytes + (uint32_t)i * (kChunk * 4u));
                }
                if (nch > kWin) {
                    // lane (li, gg): the partial sum of row li from bulk warp gg of this group
                    mbar_wait(pbar + 8u * j, 0u);
                    float p = 0.f;                      // lane 8 li carries row li's partial sum into the reduction
                    if ((lane & 7) == 0)
                        asm volatile("ld.shared.f32 %0, [%1];" : "=f"(p)
                                     : "r"(part + 16u * (uint32_t)((j % kPartDepth) * qmax + gamma) + 4u * (uint32_t)li));
#pragma unroll
                    for (int i = 0; i < kQuad; ++i) acc[i] = (i == li) ? p : 0.f;
                }
                // the window's older chunks (full ones): their blocks are at most j - 2, normally long there
#pragma unroll 1
                for (int w = max(0, kWin - nch); w < kWin - 1; ++w) {
                    const int c = nch - kWin + w;
                    const int need = block_of(c * kChunk + kChunk - 1);
                    while (ready <= need) { mbar_wait(ubar + 8u * ready, 0u); ++ready; }
                    const float4 uv = lds_f4(us + 4u * (uint32_t)(c * kChunk + lane * 4));
#pragma unroll
                    for (int i = 0; i < kQuad; ++i) {
                        const float4 gv = lds_f4(sbase + (uint32_t)w * kUnitBytes + (uint32_t)i * (kChunk * 4u));
                        acc[i] = fmaf(gv.x, uv.x, acc[i]);
                        acc[i] = fmaf(gv.y, uv.y, acc[i]);
                        acc[i] = fmaf(gv.z, uv.z, acc[i]);
                        acc[i] = fmaf(gv.w, uv.w, acc[i]);
                    }
                }
                REC_TRACE(8 + 4 * j);
                // every block the newest chunk touches must have landed HERE (completion of a later block in
                // another CTA says nothing about what has reached this one)
                ready = max(ready, block_of(cl * kChunk));
                while (ready < j) { mbar_wait(ubar + 8u * ready, 0u); ++ready; }
                REC_TRACE(9 + 4 * j);
                if (mine) {
                    const float4 uv = lds_f4(us + 4u * (uint32_t)(cl * kChunk + lane * 4));
#pragma unroll
                    for (int i = 0; i < kQuad; ++i) {
                        acc[i] = fmaf(gl[i].x, uv.x, acc[i]);
                        acc[i] = fmaf(gl[i].y, uv.y, acc[i]);
                        acc[i] = fmaf(gl[i].z, uv.z, acc[i]);
                        acc[i] = fmaf(gl[i].w, uv.w, acc[i]);
                    }
                }
            }
            const float tot = (j > 0) ? quad_reduce(acc, lane) : 0.f;       // lane l: row l >> 3
            const float zz = fmaf(-alpha, tot, rr);
            const float uu = lprime_chain<LOSS>(zz, yy);
            if (j + 1 < s || fg.Y) {                     // (the fused update needs the last block everywhere too)
                const float u0 = __shfl_sync(0xffffffffu, uu, 0), u1 = __shfl_sync(0xffffffffu, uu, 8);
                const float u2 = __shfl_sync(0xffffffffu, uu, 16), u3 = __shfl_sync(0xffffffffu, uu, 24);
                if (lane < ndst) st_async_v4(rem_us + 4u * (uint32_t)row, u0, u1, u2, u3, rem_ubar + 8u * (uint32_t)j);
            }
            REC_TRACE(10 + 4 * j);
            if ((lane & 7) == 0) {
                z[row + li] = zz;
                u[row + li] = uu;
            }
            if (j > 0) prefetch_step();                 // refills the slot consumed one step ago
            REC_TRACE(11 + 4 * j);
            rr = rr_next;
            yy = yy_next;
        }
    }
    else if (is_bulk) {
        // ===== bulk warp: every 128-column chunk of a step's rows but the newest kWin =====
        // These columns belong to blocks that landed (kWin - 1) * 128 / b hops ago, so a bulk warp can be several
        // steps ahead of the chain; it is bound by its own issue rate and the SM's L2 bandwidth.
        const int g = brank;
        const int nw = nbulk / qpc;                     // bulk warps per owned group
        const int gamma = g / nw, widx = g % nw;
        // Warp widx of a row group takes WHOLE steps j = 1 + widx, 1 + widx + nw, ...: all bulk chunks of the step,
        // one reduction and one hand-over per step (splitting every step over all warps cost a 6-shuffle reduction,
        // a barrier arrive and the loop set-up per 2-3 units). It has nw hops to finish a step.
        const uint32_t ring = base + L.bring + (uint32_t)(g * kDepth) * kUnitBytes + (uint32_t)lane * 16u;
        const float *gbase = G + (int64_t)(kQuad * (crank + gamma * C)) * ldg + lane * 4;   // + j b ldg + c * 128
        int pj = 1 + widx, pc = 0, pslot = 0;           // next unit to prefetch
        const int64_t step_stride = (int64_t)b * ldg;   // floats between the same row of consecutive blocks
        const float *prow = gbase + (int64_t)pj * step_stride;   // row group of block pj, column 0
        const float *psrc = prow;                       // ... chunk pc
        auto cursor_norm = [&]() {
            while (pj < s && pc >= num_chunks(pj, b) - kWin) { pj += nw; pc = 0; prow += nw * step_stride; psrc = prow; }
        };
        auto prefetch_unit = [&]() {
            if (pj < s) {
                const uint32_t dst = ring + (uint32_t)pslot * kUnitBytes;
                const float *src = psrc;
#pragma unroll
                for (int i = 0; i < kQuad; ++i) {
                    cp_async16_hint(dst + (uint32_t)i * (kChunk * 4u), src, pol_g);
                    src += ldg;
                }
                pc += 1;
                psrc += kChunk;
                cursor_norm();
            }
            cp_async_commit();
            pslot = (pslot + 1 == kDepth) ? 0 : pslot + 1;
        };
        cursor_norm();
#pragma unroll 1
        for (int i = 0; i < kDepth - 1; ++i) prefetch_unit();

        __syncthreads();
        cluster_sync_all();

        int slot = 0, ready = 0;
#pragma unroll 1
        for (int j = 1 + widx; j < s; j += nw) {
            const int nb = num_chunks(j, b) - kWin;
            if (nb <= 0) continue;
            REC_TRACE_B(6000 + 4 * j);
            float acc[kQuad] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll 1
            for (int c = 0; c < nb; ++c) {
                cp_async_wait<kDepth - 2>();
                float4 gv[kQuad];
#pragma unroll
                for (int i = 0; i < kQuad; ++i) gv[i] = lds_f4(ring + (uint32_t)slot * kUnitBytes + (uint32_t)i * (kChunk * 4u));
                slot = (slot + 1 == kDepth) ? 0 : slot + 1;
                const int need = block_of(c * kChunk + kChunk - 1);         // newest block this chunk touches
                while (ready <= need) { mbar_wait(ubar + 8u * ready, 0u); ++ready; }
                const float4 uv = lds_f4(us + 4u * (uint32_t)(c * kChunk + lane * 4));
#pragma unroll
                for (int i = 0; i < kQuad; ++i) {
                    acc[i] = fmaf(gv[i].x, uv.x, acc[i]);
                    acc[i] = fmaf(gv[i].y, uv.y, acc[i]);
                    acc[i] = fmaf(gv[i].z, uv.z, acc[i]);
                    acc[i] = fmaf(gv[i].w, uv.w, acc[i]);
                }
                prefetch_unit();
            }
            const float tot = quad_reduce(acc, lane);
            if ((lane & 7) == 0)
                asm volatile("st.shared.f32 [%0], %1;"
                             ::"r"(part + 16u * (uint32_t)((j % kPartDepth) * qmax + gamma) + 4u * (uint32_t)li), "f"(tot) : "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(pbar + 8u * j);
            REC_TRACE_B(6001 + 4 * j);
        }
    } else {
        __syncthreads();
        cluster_sync_all();
    }
    cp_async_wait<0>();
    if (late_trigger & 1) pdl_trigger();
    REC_TRACE(2);
    if (fg.Y) {
        // all of u is in this CTA's shared memory once every block's barrier has completed
        for (int k = threadIdx.x; k < s; k += kThreads) mbar_wait(ubar + 8u * k, 0u);
        __syncthreads();                                // ... and the rings are free: they become reduction buffers
        fused_update_tail(fg, reinterpret_cast<const float *>(rs_smem + L.u), rs_smem + L.cring, s, b, alpha, C, crank);
        REC_TRACE(3);
        __syncthreads();
        stamp_end(stamp);
        return;
    }
    __syncthreads();
    cluster_sync_all();                                 // no CTA leaves while others may still store into it
    REC_TRACE(3);
    stamp_end(stamp);
}

int stream_cluster_for(int b, int cluster_max);
constexpr int kStreamSmemCap = 227 * 1024;              // sm_100: opt-in shared memory per CTA

int stream_smem_bytes(int s, int b, int cluster_max)
{
    const int max_optin = kStreamSmemCap;
    const int c = stream_cluster_for(b, cluster_max);
    const int need = (int)stream_layout(s, b, (b / kQuad + c - 1) / c).total;
    return need <= max_optin ? need : 0;
}

// Cluster size for block size b: the largest power of two <= min(cluster_max, b / 4), so that every CTA owns
// at least one row group.
int stream_cluster_for(int b, int cluster_max)
{
    int c = 1;
    while (2 * c <= cluster_max && 2 * c <= b / kQuad) c *= 2;
    return c;
}

template <int LOSS>
cudaError_t launch_stream(cudaStream_t st, const float *G, int32_t ldg, const float *r, const float *yI, int32_t s,
                          int32_t b, float alpha, float *z, float *u, int cluster_max, const FusedGrad &fg, int late_trigger)
{
    const int smem = stream_smem_bytes(s, b, cluster_max);
    if (smem == 0) return cudaErrorInvalidConfiguration;
    auto kern = recurrence_stream_kernel<LOSS>;
    const int cluster = stream_cluster_for(b, cluster_max);
    return launch_pdl(kern, dim3(cluster), dim3(kThreads), (size_t)smem, st, cluster, G, ldg, r, yI, s, b, alpha, z, u, fg, g_stamp, late_trigger);
}

}  // namespace

cudaError_t recurrence_stream_configure()
{
    cudaError_t e = cudaSuccess;
    auto set = [&](auto kern) {
        if (e == cudaSuccess) e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kStreamSmemCap);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    };
    set(recurrence_stream_kernel<CASGD_LOGISTIC>);
    set(recurrence_stream_kernel<CASGD_LINEAR>);
    set(recurrence_stream_kernel<CASGD_POISSON>);
    return e;
}

// Can the stream kernel run this shape in a cluster of at most `cluster` CTAs?
bool recurrence_stream_ok(int32_t s, int32_t b, int32_t ldg, int cluster)
{
    if (cluster <= 0 || b % 4 != 0 || ldg % 4 != 0 || s < 2) return false;
    // part[] slots are recycled every kPartDepth steps with no back-pressure: a bulk warp's last chunk of step J ends up
    // to 2 * kChunk columns before column J * b, so it can run 2 * kChunk / b blocks ahead of the chain. That lead plus
    // the kCritPer steps the critical warps have in flight must stay below kPartDepth (b = 4: 64 blocks -- too many).
    if (2 * kChunk / b + kCritPer >= kPartDepth) return false;
    const int c = stream_cluster_for(b, cluster);
    if ((b / kQuad + c - 1) / c > kMaxQuadsPerCta) return false;
    return stream_smem_bytes(s, b, cluster) > 0;
}

// Can the streaming kernel also do the outer update of this step (small Y)?
bool recurrence_stream_fuses_update(int32_t s, int32_t b, int32_t ldy, int cluster_max)
{
    const int cluster = stream_cluster_for(b, cluster_max);
    // measured: worth it while a CTA's slice of Y stays below ~136 KB (poisson-synth s=32: 131 KB per CTA, 32.1 -> 30.4 us;
    // epsilon-shaped s=16 on 8 CTAs: 256 KB per CTA, 34.7 -> 36.9 us)
    const StreamLayout L = stream_layout(s, b, (b / kQuad + cluster - 1) / cluster);
    const int64_t buffers = (int64_t)kThreads * 8 * 4 + (int64_t)cluster * ldy * 4;      // red + CTA 0's gbuf, over the rings
    return ldy <= kFgMaxLdy && (int64_t)s * b * ldy * 2 <= (int64_t)136 * 1024 * cluster && buffers <= (int64_t)(L.total - L.cring);
}

int launch_recurrence_stream(cudaStream_t st, const float *G, int32_t ldg, const float *r, const float *yI, int32_t s,
                             int32_t b, float alpha, int loss, float *z, float *u, int cluster, const FusedUpdate *fu,
                             int late_trigger)
{
    FusedGrad fg{};
    if (fu) fg = FusedGrad{fu->Y, fu->ldy, fu->n, fu->x, fu->ind, fu->xbf, fu->split_ld, fu->r_fused};
    cudaError_t e = loss == CASGD_LOGISTIC ? launch_stream<CASGD_LOGISTIC>(st, G, ldg, r, yI, s, b, alpha, z, u, cluster, fg, late_trigger)
                  : loss == CASGD_LINEAR  ? launch_stream<CASGD_LINEAR>(st, G, ldg, r, yI, s, b, alpha, z, u, cluster, fg, late_trigger)
                                          : launch_stream<CASGD_POISSON>(st, G, ldg, r, yI, s, b, alpha, z, u, cluster, fg, late_trigger);
    return e == cudaSuccess ? 1 : -1;
}

#ifdef CASGD_REC_TRACE
extern "C" int casgd_rec_trace_dump(long long *dst_host, int n)
{
    cudaDeviceSynchronize();
    return (int)cudaMemcpyFromSymbol(dst_host, g_rec_trace, sizeof(long long) * (size_t)n);
}
#endif

}  // namespace casgd

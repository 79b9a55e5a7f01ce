// mini_step.cu -- whole outer iterations of Alg. 1 in ONE persistent launch, for steps so small
// that they are pure latency (the paper's own answer to launch latency is CUDA graphs, L278):
// BASELINE.json:configs[0] (sb = 64, n = 64), configs[1] at s = 1 and 4, configs[4] at s = 1 -- a step of a few KB that
// the kernel-per-stage path runs in 7-12 us of launch and drain.
//
// One CTA keeps everything of the chain on chip: the FP32 master x lives in shared memory for all n_steps iterations
// of the call; per iteration
//   gather      Y = A[I,:], y_I (line 2) by 16-byte cp.async into one of TWO shared-memory stages -- the rows of
//               iteration t + 1 (and the indices of t + 2) are in flight while iteration t computes;
//   margin      r = Y bf16(x) (line 3; FP32 x itself with CASGD_OPT_MARGIN_SPLIT), a lane group per row;
//   Gram        the strict block-lower G (line 4, L180) with mma.sync.m16n8k16 BF16 -> FP32 straight from the row-major
//               stage (G = Y Y^T needs no transposed operand) -- at most a few thousand MMAs: not tcgen05 territory,
//               there is no tile here worth a TMEM allocation and a descriptor;
//   recurrence  lines 6-15 in FP32 (L236), a warp per row, one __syncthreads per inner step;
//   update      g = Y^T u, x <- x - alpha g (lines 16-17), column sums over lane groups and warps in a fixed order.
// The last iteration's Y, y_I, G, r, z, u go to the context's workspaces (casgd_debug_export); x and its BF16 shadow
// are written back at the end. Same arithmetic classes as the big kernels (exact BF16 products, FP32 accumulation).
#include "common.cuh"
#include "rec_cluster.cuh"                  // lprime_chain

namespace casgd {

namespace {

constexpr int kMsMaxThreads = 512, kMsMaxWarps = 16;    // the launch picks 128 .. 512 threads
constexpr int kMsRedFloats = 4096;                      // gradient partial sums: at most 16 parts x ldy floats

struct MiniParams {
    const uint16_t *A;
    int64_t lda, m;
    const float *y;
    const int32_t *idx;                 // n_steps * s*b indices
    int64_t n_steps;
    int32_t n, ldy, s, b, exact_margin;
    float alpha;
    float *x;
    uint16_t *xbf;
    int32_t ldxb, split;
    uint16_t *Y;                        // exports of the last iteration
    float *yI, *G, *r, *z, *u;
    int32_t ldg;
    int *err_flag;
    unsigned long long *stamp;
};

// Byte offsets into dynamic shared memory. Two stages of Y, of the labels and of the indices: stage q at base + q * stride
// (scalars, not arrays indexed at run time: those end up in local memory, on every access of every phase).
struct MiniLayout {
    uint32_t x, xm, r, z, u, yl, yl_stride, idx, idx_stride, gl, red, Y, Y_stride, total;
    int32_t ldys, sbp;                  // row stride of a Y stage in elements (16-byte multiple, staggered banks); rows incl. padding
};

__host__ __device__ inline MiniLayout mini_layout(int n, int s, int b)
{
    MiniLayout L;
    const int sb = s * b;
    L.sbp = (sb + 15) & ~15;
    L.ldys = ((n + 15) & ~15) + 8;
    uint32_t o = 0;
    auto take = [&](uint32_t bytes) { const uint32_t at = o; o += (bytes + 15u) & ~15u; return at; };
    L.x = take(4u * (uint32_t)n);
    L.xm = take(4u * (uint32_t)((n + 7) & ~7));           // the margin's view of x: bf16-rounded (or x itself), zero-padded
    L.r = take(4u * sb); L.z = take(4u * sb); L.u = take(4u * sb);
    L.yl_stride = (4u * sb + 15u) & ~15u;  L.yl = take(2u * L.yl_stride);
    L.idx_stride = L.yl_stride;            L.idx = take(2u * L.idx_stride);
    L.gl = take(2u * (uint32_t)b * b * s * (s - 1));     // b^2 s (s-1) / 2 floats
    L.red = take(4u * kMsRedFloats);
    L.Y_stride = (2u * (uint32_t)L.sbp * L.ldys + 15u) & ~15u;
    L.Y = take(2u * L.Y_stride);
    L.total = o;
    return L;
}

__device__ __forceinline__ void cp_async16_ms(uint32_t dst, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4_ms(uint32_t dst, const void *src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void mma_bf16_16816(float (&c)[4], const uint32_t (&a)[4], const uint32_t (&bq)[2])
{
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(bq[0]), "r"(bq[1]));
}
__device__ __forceinline__ float bf16_round(float v) { return __bfloat162float(__float2bfloat16_rn(v)); }

#ifdef CASGD_MINI_TRACE
__device__ long long g_mini_trace[64];
#define MT(i) do { if (tid == 0 && step == 8) g_mini_trace[i] = clock64(); } while (0)
#else
#define MT(i) do { } while (0)
#endif

// The kernel is kept SMALL on purpose: every phase runs once per iteration, so its instructions are fetched once per
// iteration; a first version (runtime loss switch inlined twice, arrays of stage offsets in local memory, divisions by
// run-time values in the copy loops: 4096 instructions = 64 KB, twice the instruction cache) spent 12 000 cycles on an
// iteration that needs a few hundred FMAs. One instantiation per loss; outer loops not unrolled; power-of-two lane groups.
template <int LOSS>
__global__ void __launch_bounds__(kMsMaxThreads, 1)
mini_step_kernel(const MiniParams p)
{
    extern __shared__ __align__(128) unsigned char ms_smem[];
    pdl_trigger();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthr = blockDim.x, nwarp = nthr >> 5;
    const int s = p.s, b = p.b, sb = s * b, n = p.n, ldy = p.ldy;
    const MiniLayout L = mini_layout(n, s, b);
    const int ldys = L.ldys;
    float *xs = reinterpret_cast<float *>(ms_smem + L.x);
    float *xm = reinterpret_cast<float *>(ms_smem + L.xm);
    float *rs = reinterpret_cast<float *>(ms_smem + L.r);
    float *zs = reinterpret_cast<float *>(ms_smem + L.z);
    float *us = reinterpret_cast<float *>(ms_smem + L.u);
    float *gl = reinterpret_cast<float *>(ms_smem + L.gl);
    float *red = reinterpret_cast<float *>(ms_smem + L.red);
    const uint32_t smem0 = (uint32_t)__cvta_generic_to_shared(ms_smem);

    // both Y stages start as zeros: the K padding (columns n .. ldys) and the row padding (rows sb .. sbp) stay zero
#pragma unroll 1
    for (uint32_t o = L.Y + 16u * tid; o < L.total; o += 16u * nthr)
        *reinterpret_cast<uint4 *>(ms_smem + o) = make_uint4(0u, 0u, 0u, 0u);
    pdl_wait();                                         // x and the index buffer come from earlier work on the stream
    stamp_begin(p.stamp);
#pragma unroll 1
    for (int k = tid; k < ldy; k += nthr) {
        const float t = k < n ? p.x[k] : 0.f;
        if (k < n) xs[k] = t;
        xm[k] = p.exact_margin ? t : bf16_round(t);
    }
    if (tid < sb) {                                     // (sb <= 512: one index per thread and stage)
        reinterpret_cast<int32_t *>(ms_smem + L.idx)[tid] = p.idx[tid];
        if (p.n_steps > 1) reinterpret_cast<int32_t *>(ms_smem + L.idx + L.idx_stride)[tid] = p.idx[sb + tid];
    }
    __syncthreads();

    // gather (line 2): 16-byte cp.async pieces, CH lanes side by side on a row. (One cp.async.bulk per row on an
    // mbarrier, issued by the row's thread, measured slower -- n = 18, b = 64: 2.4 against 1.7 us per iteration, also
    // with four stages and rows three iterations ahead: the few issuing threads become the critical path of the CTA.)
    const int chunks = ldy >> 3;                        // 16-byte pieces of a gathered row
    int CH = 1, chs = 0;                                // lanes side by side on a row: a power of two >= chunks
    while (CH < chunks) { CH <<= 1; ++chs; }
    const int csub = tid & (CH - 1), crow = tid >> chs, crows = nthr >> chs;
    auto issue_gather = [&](int64_t step) {
        const uint32_t q = (uint32_t)(step & 1);
        const int32_t *I = reinterpret_cast<const int32_t *>(ms_smem + L.idx + q * L.idx_stride);
        const uint32_t ybase = L.Y + q * L.Y_stride;
        if (csub < chunks) {
#pragma unroll 1
            for (int row = crow; row < sb; row += crows) {
                const int64_t src = I[row];
                const uint32_t off = ybase + 2u * (uint32_t)(row * ldys + csub * 8);
                if (src >= 0 && src < p.m) cp_async16_ms(smem0 + off, p.A + src * p.lda + csub * 8);
                else *reinterpret_cast<uint4 *>(ms_smem + off) = make_uint4(0u, 0u, 0u, 0u);
            }
        }
        if (tid < sb) {
            const int64_t src = I[tid];
            const uint32_t off = L.yl + q * L.yl_stride + 4u * (uint32_t)tid;
            if (src >= 0 && src < p.m) cp_async4_ms(smem0 + off, p.y + src);
            else { *reinterpret_cast<float *>(ms_smem + off) = 0.f; flag_index_error(p.err_flag); }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    if (p.n_steps > 0) issue_gather(0);

    int LG = 1, lgs = 0;                                // margin: lanes side by side on a row (<= 32)
    while (LG < chunks && LG < 32) { LG <<= 1; ++lgs; }
    const int msub = tid & (LG - 1), mrow = tid >> lgs, mrows = nthr >> lgs;
    const uint32_t inv_b = ((1u << 20) + (uint32_t)b - 1u) / (uint32_t)b;    // floor(i / b) = i * inv_b >> 20 for i b < 2^20

#pragma unroll 1
    for (int64_t step = 0; step < p.n_steps; ++step) {
        const uint32_t q = (uint32_t)(step & 1);
        const bool last = step + 1 == p.n_steps;
        MT(0);
        // rows of the next iteration; indices of the one after it (stored at the bottom of this iteration)
        if (!last) issue_gather(step + 1); else asm volatile("cp.async.commit_group;" ::: "memory");
        MT(8);
        int32_t idx_next = 0;
        if (step + 2 < p.n_steps && tid < sb) idx_next = p.idx[(step + 2) * sb + tid];
        asm volatile("cp.async.wait_group 1;" ::: "memory");
        MT(1);
        __syncthreads();                                // this iteration's rows and labels are in shared memory
        uint16_t *Ys = reinterpret_cast<uint16_t *>(ms_smem + L.Y + q * L.Y_stride);
        const float *yl = reinterpret_cast<const float *>(ms_smem + L.yl + q * L.yl_stride);
        if (n & 7) {                                    // A's own padding may hold anything: Y's pad columns are zero
            if (tid < sb)
                for (int c = n; c < ldy; ++c) Ys[tid * ldys + c] = 0;
            __syncthreads();
        }

        MT(2);
        // ---- margin (line 3): a group of LG lanes per row, 8 columns per lane and pass
#pragma unroll 1
        for (int i0 = 0; i0 < sb; i0 += mrows) {        // (uniform trip count: every lane takes part in the shuffles)
            const int i = i0 + mrow;
            float acc = 0.f, acc2 = 0.f;
#pragma unroll 1
            for (int c = msub; c < chunks && i < sb; c += LG) {
                const uint4 v = *reinterpret_cast<const uint4 *>(Ys + i * ldys + c * 8);
                const float4 xa = *reinterpret_cast<const float4 *>(xm + c * 8), xb = *reinterpret_cast<const float4 *>(xm + c * 8 + 4);
                acc = fmaf(bf16lo(v.x), xa.x, acc); acc2 = fmaf(bf16hi(v.x), xa.y, acc2);
                acc = fmaf(bf16lo(v.y), xa.z, acc); acc2 = fmaf(bf16hi(v.y), xa.w, acc2);
                acc = fmaf(bf16lo(v.z), xb.x, acc); acc2 = fmaf(bf16hi(v.z), xb.y, acc2);
                acc = fmaf(bf16lo(v.w), xb.z, acc); acc2 = fmaf(bf16hi(v.w), xb.w, acc2);
            }
            acc += acc2;
            MT(10);
            for (int o = LG >> 1; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
            MT(11);
            if (msub == 0 && i < sb) {
                rs[i] = acc;
                zs[i] = acc;                            // (s > 1: the recurrence starts from z = r)
                if (s == 1) us[i] = lprime_chain<LOSS>(acc, yl[i]);
            }
        }

        MT(3);
        // ---- Gram (line 4): 16 x 8 tiles of the strict block-lower part, mma.sync from the row-major stage; the tiles
        // of all row tiles form ONE job list dealt to the warps. G lands TRANSPOSED inside each b x b block --
        // entry (i, k), block(i) = jr > block(k) = jc, at  b^2 jr (jr-1) / 2 + jc b^2 + (k - jc b) b + (i - jr b) --
        // so that the recurrence below reads it with consecutive threads on consecutive words.
        if (s > 1) {
            const int g = lane >> 2, t4 = lane & 3;
            const int TR = L.sbp >> 4, ksteps = (ldys - 8) >> 4;
            int first = 0, job = warp;                  // jobs before this row tile; this warp's next job
#pragma unroll 1
            for (int tr = 0; tr < TR; ++tr) {           // (a row tile inside block 0 has no columns: ntc = 0)
                const int row_hi = min(tr * 16 + 15, sb - 1);
                const int ntc = ((int)((uint32_t)row_hi * inv_b >> 20) * b + 7) >> 3;      // 8-column tiles that hold a block below some row of the tile
#pragma unroll 1
                for (; job < first + ntc; job += nwarp) {
                    const int tc = job - first;
                    float c[4] = {0.f, 0.f, 0.f, 0.f};
                    const uint16_t *arow0 = Ys + (tr * 16 + g) * ldys + 2 * t4, *arow1 = arow0 + 8 * ldys;
                    const uint16_t *brow = Ys + (tc * 8 + g) * ldys + 2 * t4;
#pragma unroll 2
                    for (int ks = 0; ks < ksteps; ++ks) {
                        uint32_t a[4], bq[2];
                        a[0] = *reinterpret_cast<const uint32_t *>(arow0 + ks * 16);
                        a[1] = *reinterpret_cast<const uint32_t *>(arow1 + ks * 16);
                        a[2] = *reinterpret_cast<const uint32_t *>(arow0 + ks * 16 + 8);
                        a[3] = *reinterpret_cast<const uint32_t *>(arow1 + ks * 16 + 8);
                        bq[0] = *reinterpret_cast<const uint32_t *>(brow + ks * 16);
                        bq[1] = *reinterpret_cast<const uint32_t *>(brow + ks * 16 + 8);
                        mma_bf16_16816(c, a, bq);
                    }
                    // rows i0, i0 + 8 and columns k0, k0 + 1 of this lane: block numbers once per row and column
                    const int i0 = tr * 16 + g, k0 = tc * 8 + 2 * t4, bb = b * b;
                    int jrow[2], jcol[2], roff[2], coff[2];
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        jrow[h] = (int)((uint32_t)(i0 + 8 * h) * inv_b >> 20);
                        jcol[h] = (int)((uint32_t)(k0 + h) * inv_b >> 20);
                        roff[h] = (bb * jrow[h] * (jrow[h] - 1)) / 2 + (i0 + 8 * h - jrow[h] * b);
                        coff[h] = jcol[h] * bb + (k0 + h - jcol[h] * b) * b;
                    }
#pragma unroll
                    for (int e = 0; e < 4; ++e)
                        if (i0 + 8 * (e >> 1) < sb && jcol[e & 1] < jrow[e >> 1]) gl[roff[e >> 1] + coff[e & 1]] = c[e];
                }
                first += ntc;
            }
        }
        __syncthreads();
        MT(4);

        // ---- recurrence (lines 6-15), right-looking, a THREAD per row (s b <= the threads): the margin left z = r;
        // per inner step the rows of block j apply l', one barrier, and every later row takes block j's b columns off
        // its own z -- the rows of block j + 1 are then final without another barrier.
        if (s > 1) {
            const int jr = tid / b, il = tid - jr * b;  // this thread's row: block and row inside it
            const float *gmine = gl + (b * b * jr * (jr - 1)) / 2 + il;
            float zmine = tid < sb ? zs[tid] : 0.f;
#pragma unroll 1
            for (int j = 0; j < s; ++j) {
                if (tid < sb && jr == j) {
                    zs[tid] = zmine;
                    us[tid] = lprime_chain<LOSS>(zmine, yl[tid]);
                }
                __syncthreads();
                if (tid < sb && jr > j) {
                    const float *gcol = gmine + j * b * b, *uj = us + j * b;
                    float a0 = 0.f, a1 = 0.f;
                    int k = 0;
#pragma unroll 4
                    for (; k + 1 < b; k += 2) {
                        a0 = fmaf(gcol[k * b], uj[k], a0);
                        a1 = fmaf(gcol[(k + 1) * b], uj[k + 1], a1);
                    }
                    if (k < b) a0 = fmaf(gcol[k * b], uj[k], a0);
                    zmine = fmaf(-p.alpha, a0 + a1, zmine);
                }
            }
        }

        MT(5);
        // ---- update (lines 16-17): g = Y^T u by lane groups (8 columns per thread), rows split over the groups; the
        // groups of a warp meet by shuffles, the 16 warps through shared memory, in a fixed order
        {
            float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
            if (csub < chunks)
#pragma unroll 1
                for (int i = crow; i < sb; i += crows) {
                    const uint4 v = *reinterpret_cast<const uint4 *>(Ys + i * ldys + csub * 8);
                    const float uu = us[i];
                    acc[0] = fmaf(bf16lo(v.x), uu, acc[0]); acc[1] = fmaf(bf16hi(v.x), uu, acc[1]);
                    acc[2] = fmaf(bf16lo(v.y), uu, acc[2]); acc[3] = fmaf(bf16hi(v.y), uu, acc[3]);
                    acc[4] = fmaf(bf16lo(v.z), uu, acc[4]); acc[5] = fmaf(bf16hi(v.z), uu, acc[5]);
                    acc[6] = fmaf(bf16lo(v.w), uu, acc[6]); acc[7] = fmaf(bf16hi(v.w), uu, acc[7]);
                }
#pragma unroll 1
            for (int o = CH; o < 32; o <<= 1)
#pragma unroll
                for (int e = 0; e < 8; ++e) acc[e] += __shfl_xor_sync(0xffffffffu, acc[e], o);
            // partial sums that remain: one per warp when CH <= 32, one per row group otherwise (then <= 16 groups)
            const int nred = CH <= 32 ? nwarp : crows, ridx = CH <= 32 ? warp : crow;
            if (csub < chunks && (CH > 32 || lane < CH)) {
#pragma unroll
                for (int e = 0; e < 8; ++e) red[ridx * ldy + csub * 8 + e] = acc[e];
            }
            __syncthreads();
#pragma unroll 1
            for (int col = tid; col < n; col += nthr) {
                float gsum = 0.f;
#pragma unroll 4
                for (int r2 = 0; r2 < nred; ++r2) gsum += red[r2 * ldy + col];
                const float xn = fmaf(-p.alpha, gsum, xs[col]);
                xs[col] = xn;
                xm[col] = p.exact_margin ? xn : bf16_round(xn);
            }
        }

        MT(6);
        if (last) {
            // the intermediates casgd_debug_export serves
            if (csub < chunks)
#pragma unroll 1
                for (int row = crow; row < sb; row += crows)
                    *reinterpret_cast<uint4 *>(p.Y + (int64_t)row * ldy + csub * 8) = *reinterpret_cast<const uint4 *>(Ys + row * ldys + csub * 8);
            if (tid < sb) { p.yI[tid] = yl[tid]; p.r[tid] = rs[tid]; p.z[tid] = zs[tid]; p.u[tid] = us[tid]; }
#pragma unroll 1
            for (int i = b + warp; i < sb; i += nwarp) {
                const int j = i / b;
                const float *gt = gl + (b * b * j * (j - 1)) / 2 + (i - j * b);      // (k, i) of the row block, transposed blocks
#pragma unroll 1
                for (int k = lane; k < j * b; k += 32) p.G[(int64_t)i * p.ldg + k] = gt[k * b];
            }
        }
        if (step + 2 < p.n_steps && tid < sb) reinterpret_cast<int32_t *>(ms_smem + L.idx + q * L.idx_stride)[tid] = idx_next;
        __syncthreads();                                // x, the stage and the vectors are free for the next iteration
        MT(7);
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
#pragma unroll 1
    for (int k = tid; k < n; k += nthr) {
        const float xn = xs[k];
        p.x[k] = xn;
        store_shadow(p.xbf, p.split ? p.ldxb : 0, k, xn);
    }
    __syncthreads();
    stamp_end(p.stamp);
}

constexpr int kMiniSmemCap = 227 * 1024;

}  // namespace

cudaError_t mini_step_configure()
{
    cudaError_t e = cudaFuncSetAttribute(mini_step_kernel<CASGD_LOGISTIC>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMiniSmemCap);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(mini_step_kernel<CASGD_LINEAR>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMiniSmemCap);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(mini_step_kernel<CASGD_POISSON>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMiniSmemCap);
    return e;
}

// Does the one-launch kernel take this shape? Everything of an iteration (two Y stages, the packed strict block-lower
// G, the vectors) must fit one CTA's shared memory, and the Gram and the chain must be small enough for one SM.
bool mini_step_ok(int32_t n, int32_t ldy, int32_t s, int32_t b, bool any_fit)
{
    const int64_t sb = (int64_t)s * b;
    if (n < 1 || n > 2048 || sb > kMsMaxThreads || ldy != ((n + 7) & ~7)) return false;   // (one index per thread)
    if ((int64_t)b * b * s * (s - 1) * 2 > 160 * 1024) return false;
    // gradient partial sums: 16 warps (row groups of <= 32 lanes) or 512 / CH parts, times ldy floats
    int CH = 1;
    while (CH < ldy / 8) CH <<= 1;
    const int nred = CH <= 32 ? kMsMaxWarps : kMsMaxThreads / CH;
    if ((int64_t)nred * ldy > kMsRedFloats) return false;
    if (mini_layout(n, s, b).total > (uint32_t)kMiniSmemCap) return false;
    // measured crossovers against the kernel-per-stage path (us per iteration): s = 1 wins up to 32 KB of rows per step
    // (n = 18, b = 64: 1.4 against 7.2; n = 128, b = 128: 4.0 against 6.3; n = 128, b = 256: 9.0 against 7.2) and for
    // rows of <= 128 bytes at any b (n = 64, b = 512: 5.8 against 10.3); steps beyond 4 KB with rows of >= 128 bytes go to the
    // cluster kernel first (s1_cluster.cu; n = 256, b = 64: 1.9 against 5.2 here). s > 1 wins while Gram and chain are tiny
    // (n = 64, s = 4, b = 16: 3.7 against 8.0; n = 64, s = 8, b = 16: 8.5 against 9.4; n = 128, s = 4, b = 32: 9.1 against
    // 8.0; n = 512, s = 2, b = 32: 10.7 against 8.0)
    if (any_fit) return true;                           // CASGD_OPT_MINI = 2: the structural limits only
    if (s == 1) return (int64_t)b * ldy * 2 <= 32 * 1024 || ldy <= 64;
    const int64_t macs = (int64_t)((n + 15) & ~15) * b * b * s * (s - 1) / 2;
    return sb <= 128 && macs <= (460ll << 10) && (int64_t)s * ((b + kMsMaxWarps - 1) / kMsMaxWarps) <= 16;
}

int launch_mini_steps(cudaStream_t st, const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n, int32_t ldy,
                      const int32_t *idx, int64_t n_steps, int32_t s, int32_t b, float alpha, int loss, int exact_margin,
                      float *x, uint16_t *xbf, int32_t ldxb, int split, uint16_t *Y, float *yI, float *G, int32_t ldg, float *r,
                      float *z, float *u, int *err_flag)
{
    MiniParams p;
    p.A = A; p.lda = lda; p.m = m; p.y = y; p.idx = idx; p.n_steps = n_steps; p.n = n; p.ldy = ldy; p.s = s; p.b = b;
    p.exact_margin = exact_margin; p.alpha = alpha; p.x = x; p.xbf = xbf; p.ldxb = ldxb; p.split = split;
    p.Y = Y; p.yI = yI; p.G = G; p.r = r; p.z = z; p.u = u; p.ldg = ldg; p.err_flag = err_flag; p.stamp = g_stamp;
    const MiniLayout L = mini_layout(n, s, b);
    auto *kern = loss == CASGD_LOGISTIC ? mini_step_kernel<CASGD_LOGISTIC>
               : loss == CASGD_LINEAR  ? mini_step_kernel<CASGD_LINEAR>
                                       : mini_step_kernel<CASGD_POISSON>;
    // measured: the barriers of a small s = 1 iteration are cheaper with 8 warps (n = 18, b = 64: 1.43 against 1.68 us;
    // from 12 KB of rows on 16 warps win again), the
    // chain of s > 1 wants a warp per row of a block (n = 64, s = 4, b = 16: 5.2 us with 16 warps, 6.0 with 8)
    int threads = s == 1 && b * ldy * 2 <= 4096 ? 256 : kMsMaxThreads;
    while (threads < s * b || threads * 8 < ldy) threads <<= 1;    // one index per thread; a row's 16-byte pieces side by side
    return launch_pdl(kern, dim3(1), dim3(threads), (size_t)L.total, st, 1, p) == cudaSuccess ? 1 : -1;
}

#ifdef CASGD_MINI_TRACE
extern "C" int casgd_mini_trace_dump(long long *dst_host)
{
    cudaDeviceSynchronize();
    return (int)cudaMemcpyFromSymbol(dst_host, g_mini_trace, sizeof(long long) * 64);
}
#endif

}  // namespace casgd

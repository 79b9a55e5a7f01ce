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

namespace casgd {

namespace {

constexpr int kMsThreads = 512, kMsWarps = 16;
constexpr int kMsRedFloats = 4096;                      // gradient partial sums: <= 16 parts x ldy, ldy <= 2048 / ... (see layout)

struct MiniParams {
    const uint16_t *A;
    int64_t lda, m;
    const float *y;
    const int32_t *idx;                 // n_steps * s*b indices
    int64_t n_steps;
    int32_t n, ldy, s, b, loss, exact_margin, stages;
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

constexpr int kMsMaxStages = 4;
struct MiniLayout {                     // byte offsets into dynamic shared memory
    uint32_t x, r, z, u, yl[kMsMaxStages], idx[kMsMaxStages], gl, red, Y[kMsMaxStages], total;
    int32_t ldys, sbp;                  // row stride of a Y stage in elements (16-byte multiple, staggered banks); rows incl. padding
};

__host__ __device__ inline MiniLayout mini_layout(int n, int s, int b, int ns)
{
    MiniLayout L;
    const int sb = s * b;
    L.sbp = (sb + 15) & ~15;
    L.ldys = ((n + 15) & ~15) + 8;
    uint32_t o = 0;
    auto take = [&](uint32_t bytes) { const uint32_t at = o; o += (bytes + 15u) & ~15u; return at; };
    L.x = take(4u * (uint32_t)n);
    L.r = take(4u * sb); L.z = take(4u * sb); L.u = take(4u * sb);
    for (int q = 0; q < ns; ++q) L.yl[q] = take(4u * sb);
    for (int q = 0; q < ns; ++q) L.idx[q] = take(4u * sb);
    L.gl = take(2u * (uint32_t)b * b * s * (s - 1));     // b^2 s (s-1) / 2 floats
    L.red = take(4u * kMsRedFloats);
    for (int q = 0; q < ns; ++q) L.Y[q] = take(2u * (uint32_t)L.sbp * L.ldys);
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

__global__ void __launch_bounds__(kMsThreads, 1)
mini_step_kernel(const MiniParams p)
{
    extern __shared__ __align__(128) unsigned char ms_smem[];
    pdl_trigger();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int s = p.s, b = p.b, sb = s * b, n = p.n, ldy = p.ldy;
    const int NS = p.stages, D = NS - 1;              // Y stages; rows are gathered D iterations ahead
    const MiniLayout L = mini_layout(n, s, b, NS);
    const int ldys = L.ldys;
    float *xs = reinterpret_cast<float *>(ms_smem + L.x);
    float *rs = reinterpret_cast<float *>(ms_smem + L.r);
    float *zs = reinterpret_cast<float *>(ms_smem + L.z);
    float *us = reinterpret_cast<float *>(ms_smem + L.u);
    float *gl = reinterpret_cast<float *>(ms_smem + L.gl);
    float *red = reinterpret_cast<float *>(ms_smem + L.red);
    const uint32_t smem0 = (uint32_t)__cvta_generic_to_shared(ms_smem);

    // both Y stages start as zeros: the K padding (columns n .. ldys) and the row padding (rows sb .. sbp) stay zero
    for (uint32_t o = L.Y[0] + 16u * tid; o < L.total; o += 16u * kMsThreads)
        *reinterpret_cast<uint4 *>(ms_smem + o) = make_uint4(0u, 0u, 0u, 0u);
    pdl_wait();                                         // x and the index buffer come from earlier work on the stream
    stamp_begin(p.stamp);
    for (int k = tid; k < n; k += kMsThreads) xs[k] = p.x[k];
    for (int q = 0; q < NS; ++q)
        if (q < p.n_steps)
            for (int i = tid; i < sb; i += kMsThreads)
                reinterpret_cast<int32_t *>(ms_smem + L.idx[q])[i] = p.idx[(int64_t)q * sb + i];
    __syncthreads();

    const int chunks = ldy >> 3;                        // 16-byte pieces of a gathered row
    auto issue_gather = [&](int64_t step) {
        const int buf = (int)(step % NS);
        const int32_t *I = reinterpret_cast<const int32_t *>(ms_smem + L.idx[buf]);
        for (int t = tid; t < sb * chunks; t += kMsThreads) {
            const int row = t / chunks, c = t - row * chunks;
            const int64_t src = I[row];
            const uint32_t dst = smem0 + L.Y[buf] + 2u * (uint32_t)(row * ldys + c * 8);
            if (src >= 0 && src < p.m) cp_async16_ms(dst, p.A + src * p.lda + c * 8);
            else *reinterpret_cast<uint4 *>(ms_smem + (dst - smem0)) = make_uint4(0u, 0u, 0u, 0u);
        }
        for (int i = tid; i < sb; i += kMsThreads) {
            const int64_t src = I[i];
            if (src >= 0 && src < p.m) cp_async4_ms(smem0 + L.yl[buf] + 4u * i, p.y + src);
            else { reinterpret_cast<float *>(ms_smem + L.yl[buf])[i] = 0.f; atomicOr(p.err_flag, 1); }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    for (int q = 0; q < D; ++q) {
        if (q < p.n_steps) issue_gather(q); else asm volatile("cp.async.commit_group;" ::: "memory");
    }

    for (int64_t step = 0; step < p.n_steps; ++step) {
        const int buf = (int)(step % NS);
        const bool last = step + 1 == p.n_steps;
        // rows of iteration step + D; indices of the one after that (stored at the bottom of this iteration)
        if (step + D < p.n_steps) issue_gather(step + D); else asm volatile("cp.async.commit_group;" ::: "memory");
        int32_t idx_next[4] = {0, 0, 0, 0};             // sb <= 4 * 512
        if (step + NS < p.n_steps)
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (tid + q * kMsThreads < sb) idx_next[q] = p.idx[(step + NS) * sb + tid + q * kMsThreads];
        if (D == 1) asm volatile("cp.async.wait_group 1;" ::: "memory");
        else asm volatile("cp.async.wait_group 3;" ::: "memory");
        __syncthreads();                                // this iteration's rows and labels are in shared memory
        uint16_t *Ys = reinterpret_cast<uint16_t *>(ms_smem + L.Y[buf]);
        const float *yl = reinterpret_cast<const float *>(ms_smem + L.yl[buf]);
        if (n & 7) {                                    // A's own padding may hold anything: Y's pad columns are zero
            for (int i = tid; i < sb; i += kMsThreads)
                for (int c = n; c < ldy; ++c) Ys[i * ldys + c] = 0;
            __syncthreads();
        }

        // ---- margin (line 3): a group of LG lanes per row, 8 columns per lane and pass
        {
            int LG = 1;
            while (LG < chunks && LG < 32) LG <<= 1;
            const int rows_per_pass = kMsThreads / LG, sub = tid % LG;
            for (int i0 = 0; i0 < sb; i0 += rows_per_pass) {   // (uniform trip count: every lane takes part in the shuffles)
                const int i = i0 + tid / LG;
                float acc = 0.f;
                for (int c = sub; c < chunks && i < sb; c += LG) {
                    const uint4 v = *reinterpret_cast<const uint4 *>(Ys + i * ldys + c * 8);
                    const float *xv = xs + c * 8;
                    float xe[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const float t = c * 8 + e < n ? xv[e] : 0.f;
                        xe[e] = p.exact_margin ? t : bf16_round(t);
                    }
                    acc = fmaf(bf16lo(v.x), xe[0], acc); acc = fmaf(bf16hi(v.x), xe[1], acc);
                    acc = fmaf(bf16lo(v.y), xe[2], acc); acc = fmaf(bf16hi(v.y), xe[3], acc);
                    acc = fmaf(bf16lo(v.z), xe[4], acc); acc = fmaf(bf16hi(v.z), xe[5], acc);
                    acc = fmaf(bf16lo(v.w), xe[6], acc); acc = fmaf(bf16hi(v.w), xe[7], acc);
                }
                for (int o = LG >> 1; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
                if (sub == 0 && i < sb) {
                    rs[i] = acc;
                    if (s == 1) { zs[i] = acc; us[i] = lprime_rt(p.loss, acc, yl[i]); }
                }
            }
        }

        // ---- Gram (line 4): 16 x 8 tiles of the strict block-lower part, mma.sync from the row-major stage
        if (s > 1) {
            const int g = lane >> 2, t4 = lane & 3;
            const int TR = L.sbp >> 4, ksteps = (ldys - 8) >> 4;
            for (int tr = 0; tr < TR; ++tr) {           // (a row tile inside block 0 has no columns: ntc = 0)
                const int row_hi = min(tr * 16 + 15, sb - 1);
                const int ncols = (row_hi / b) * b;     // columns [0, ncols) hold a block below the block of some row of the tile
                const int ntc = (ncols + 7) >> 3;
                for (int tc = warp; tc < ntc; tc += kMsWarps) {
                    float c[4] = {0.f, 0.f, 0.f, 0.f};
                    const uint16_t *arow0 = Ys + (tr * 16 + g) * ldys + 2 * t4, *arow1 = arow0 + 8 * ldys;
                    const uint16_t *brow = Ys + (tc * 8 + g) * ldys + 2 * t4;
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
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const int i = tr * 16 + g + (e >> 1) * 8, k = tc * 8 + 2 * t4 + (e & 1);
                        const int j = i / b;
                        if (i < sb && k < j * b) gl[(b * b * j * (j - 1)) / 2 + (i - j * b) * j * b + k] = c[e];
                    }
                }
            }
        }
        __syncthreads();

        // ---- recurrence (lines 6-15): a warp per row of block j, one barrier per inner step
        if (s > 1) {
            for (int j = 0; j < s; ++j) {
                const int len = j * b;
                const float *gblk = gl + (b * b * j * (j - 1)) / 2;
                for (int i = j * b + warp; i < (j + 1) * b; i += kMsWarps) {
                    float acc = 0.f;
                    const float *grow = gblk + (i - j * b) * len;
                    for (int k = lane; k < len; k += 32) acc = fmaf(grow[k], us[k], acc);
                    acc = warp_sum(acc);
                    if (lane == 0) {
                        const float zz = fmaf(-p.alpha, acc, rs[i]);
                        zs[i] = zz;
                        us[i] = lprime_rt(p.loss, zz, yl[i]);
                    }
                }
                __syncthreads();
            }
        }

        // ---- update (lines 16-17): g = Y^T u by lane groups (8 columns per thread), rows split over the groups; the
        // groups of a warp meet by shuffles, the 16 warps through shared memory, in a fixed order
        {
            int CH = 1;
            while (CH < chunks) CH <<= 1;               // lanes side by side on a row (power of two)
            const int c = tid % CH, part = tid / CH, parts = kMsThreads / CH;
            float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
            if (c < chunks)
                for (int i = part; i < sb; i += parts) {
                    const uint4 v = *reinterpret_cast<const uint4 *>(Ys + i * ldys + c * 8);
                    const float uu = us[i];
                    acc[0] = fmaf(bf16lo(v.x), uu, acc[0]); acc[1] = fmaf(bf16hi(v.x), uu, acc[1]);
                    acc[2] = fmaf(bf16lo(v.y), uu, acc[2]); acc[3] = fmaf(bf16hi(v.y), uu, acc[3]);
                    acc[4] = fmaf(bf16lo(v.z), uu, acc[4]); acc[5] = fmaf(bf16hi(v.z), uu, acc[5]);
                    acc[6] = fmaf(bf16lo(v.w), uu, acc[6]); acc[7] = fmaf(bf16hi(v.w), uu, acc[7]);
                }
            for (int o = CH; o < 32; o <<= 1)
#pragma unroll
                for (int e = 0; e < 8; ++e) acc[e] += __shfl_xor_sync(0xffffffffu, acc[e], o);
            // partial sums that remain: one per warp when CH <= 32, one per `part` otherwise (then parts <= 16)
            const int nred = CH <= 32 ? kMsWarps : parts, ridx = CH <= 32 ? warp : part;
            if (c < chunks && (CH > 32 || lane < CH)) {
#pragma unroll
                for (int e = 0; e < 8; ++e) red[ridx * ldy + c * 8 + e] = acc[e];
            }
            __syncthreads();
            for (int col = tid; col < n; col += kMsThreads) {
                float gsum = 0.f;
                for (int q = 0; q < nred; ++q) gsum += red[q * ldy + col];
                xs[col] = fmaf(-p.alpha, gsum, xs[col]);
            }
        }

        if (last) {
            // the intermediates casgd_debug_export serves
            for (int t = tid; t < sb * chunks; t += kMsThreads) {
                const int row = t / chunks, c = t - row * chunks;
                *reinterpret_cast<uint4 *>(p.Y + (int64_t)row * ldy + c * 8) = *reinterpret_cast<const uint4 *>(Ys + row * ldys + c * 8);
            }
            for (int i = tid; i < sb; i += kMsThreads) { p.yI[i] = yl[i]; p.r[i] = rs[i]; p.z[i] = zs[i]; p.u[i] = us[i]; }
            for (int i = b + warp; i < sb; i += kMsWarps) {
                const int j = i / b;
                const float *grow = gl + (b * b * j * (j - 1)) / 2 + (i - j * b) * j * b;
                for (int k = lane; k < j * b; k += 32) p.G[(int64_t)i * p.ldg + k] = grow[k];
            }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q)
            if (step + NS < p.n_steps && tid + q * kMsThreads < sb)
                reinterpret_cast<int32_t *>(ms_smem + L.idx[buf])[tid + q * kMsThreads] = idx_next[q];
        __syncthreads();                                // x, the stage and the vectors are free for the next iteration
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    for (int k = tid; k < n; k += kMsThreads) {
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
    return cudaFuncSetAttribute(mini_step_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kMiniSmemCap);
}

// Does the one-launch kernel take this shape? Everything of an iteration (two Y stages, the packed strict block-lower
// G, the vectors) must fit one CTA's shared memory, and the Gram and the chain must be small enough for one SM.
bool mini_step_ok(int32_t n, int32_t ldy, int32_t s, int32_t b)
{
    const int64_t sb = (int64_t)s * b;
    if (n < 1 || n > 2048 || sb > 2048 || ldy != ((n + 7) & ~7)) return false;
    if ((int64_t)b * b * s * (s - 1) * 2 > 160 * 1024) return false;
    // gradient partial sums: 16 warps (row groups of <= 32 lanes) or 512 / CH parts, times ldy floats
    int CH = 1;
    while (CH < ldy / 8) CH <<= 1;
    const int nred = CH <= 32 ? kMsWarps : kMsThreads / CH;
    if ((int64_t)nred * ldy > kMsRedFloats) return false;
    const MiniLayout L = mini_layout(n, s, b, 2);
    if (L.total > (uint32_t)kMiniSmemCap) return false;
    // measured crossovers against the kernel-per-stage path: s = 1 wins while the rows of a step are a few KB (n = 18,
    // b = 64: 2.4 against 7.2 us; n = 512, b = 64 -- 64 KB through one SM -- 8.9 against 8.0); s > 1 while Gram and chain
    // are tiny (n = 64, sb = 64: 6.1 against 8.4 us; n = 18, sb = 256: 19.2 against 9.3)
    if (s == 1) return (int64_t)b * ldy * 2 <= 16 * 1024;
    const int64_t macs = (int64_t)((n + 15) & ~15) * b * b * s * (s - 1) / 2;
    return sb <= 128 && macs <= (256ll << 10) && (int64_t)s * ((b + kMsWarps - 1) / kMsWarps) <= 16;
}

int launch_mini_steps(cudaStream_t st, const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n, int32_t ldy,
                      const int32_t *idx, int64_t n_steps, int32_t s, int32_t b, float alpha, int loss, int exact_margin,
                      float *x, uint16_t *xbf, int32_t ldxb, int split, uint16_t *Y, float *yI, float *G, int32_t ldg, float *r,
                      float *z, float *u, int *err_flag)
{
    MiniParams p;
    p.A = A; p.lda = lda; p.m = m; p.y = y; p.idx = idx; p.n_steps = n_steps; p.n = n; p.ldy = ldy; p.s = s; p.b = b;
    p.loss = loss; p.exact_margin = exact_margin; p.alpha = alpha; p.x = x; p.xbf = xbf; p.ldxb = ldxb; p.split = split;
    p.Y = Y; p.yI = yI; p.G = G; p.r = r; p.z = z; p.u = u; p.ldg = ldg; p.err_flag = err_flag; p.stamp = g_stamp;
    // rows are gathered ONE iteration ahead (two stages). Measured with four stages (three iterations ahead): no gain
    // (n = 18, b = 64, s = 1: 2.71 against 2.43 us per step) -- an iteration is bound by its own dependent phases and
    // barriers, not by the latency of the rows.
    p.stages = 2;
    const MiniLayout L = mini_layout(n, s, b, p.stages);
    return launch_pdl(mini_step_kernel, dim3(1), dim3(kMsThreads), (size_t)L.total, st, 1, p) == cudaSuccess ? 1 : -1;
}

}  // namespace casgd

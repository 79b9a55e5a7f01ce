// gradient.cu -- Alg. 1 lines 16-17 fused: g = Y^T u ; x <- x - alpha g (FP32 master);
// x_bf <- bf16_rne(x) for the next margin (L231). The paper fuses GEMV + update into one GEMM with
// alpha = eta/b, beta = 1 (L272); here it is one streaming kernel: 16-byte loads of Y, u kept FP32,
// FP32 accumulation, deterministic two-level reduction (per-CTA column sums, then the last CTA of a
// column tile adds the partials in a fixed order and applies the update).
// Also the all-FP32 s = 1 baseline (Recipe A, L99): margin + residual kernel and the same gradient
// kernel reading FP32 rows of A through the index list.
#include "common.cuh"

namespace casgd {

template <typename T> struct VecTraits;
template <> struct VecTraits<uint16_t> {            // 8 BF16 per 16-byte load
    static constexpr int kVec = 8;
    __device__ static void fma_into(float (&acc)[8], const uint4 &v, float uu)
    {
        acc[0] = fmaf(bf16lo(v.x), uu, acc[0]); acc[1] = fmaf(bf16hi(v.x), uu, acc[1]);
        acc[2] = fmaf(bf16lo(v.y), uu, acc[2]); acc[3] = fmaf(bf16hi(v.y), uu, acc[3]);
        acc[4] = fmaf(bf16lo(v.z), uu, acc[4]); acc[5] = fmaf(bf16hi(v.z), uu, acc[5]);
        acc[6] = fmaf(bf16lo(v.w), uu, acc[6]); acc[7] = fmaf(bf16hi(v.w), uu, acc[7]);
    }
};
template <> struct VecTraits<float> {               // 4 FP32 per 16-byte load
    static constexpr int kVec = 4;
    __device__ static void fma_into(float (&acc)[4], const uint4 &v, float uu)
    {
        acc[0] = fmaf(__uint_as_float(v.x), uu, acc[0]); acc[1] = fmaf(__uint_as_float(v.y), uu, acc[1]);
        acc[2] = fmaf(__uint_as_float(v.z), uu, acc[2]); acc[3] = fmaf(__uint_as_float(v.w), uu, acc[3]);
    }
};

constexpr int kGradThreads = 256;

// grid = (column tiles, row splits). Thread (cvl, rl): column vector cvl of the tile, row lane rl.
// GATHER: rows are base + idx[row]*ld (FP32 baseline), else base + row*ld (the staged Y).
template <typename T, bool GATHER, bool SHADOW>
__global__ void __launch_bounds__(kGradThreads)
gradient_update_kernel(const T *base, int64_t ld, const int32_t *idx, int64_t m, int32_t n,
                       int32_t rows, int32_t rows_per_split, int32_t CV, const float *u, float alpha,
                       float *x_direct, const StepParams *ind, uint16_t *xbf, int32_t split_ld,
                       float *partial, int32_t ldp, unsigned *counters, unsigned long long *stamp)
{
    constexpr int kVec = VecTraits<T>::kVec;
    pdl_trigger();
    pdl_wait();
    stamp_begin(stamp);
    __shared__ float red[kGradThreads * kVec];
    __shared__ bool s_last;
    const int tid = threadIdx.x;
    const int cvl = tid % CV, rl = tid / CV, RL = kGradThreads / CV;
    const int nvec = (n + kVec - 1) / kVec;
    const int cv = blockIdx.x * CV + cvl;
    const bool active = cv < nvec;
    const int r0 = blockIdx.y * rows_per_split, r1 = min(rows, r0 + rows_per_split);

    float acc[kVec];
#pragma unroll
    for (int k = 0; k < kVec; ++k) acc[k] = 0.f;
    if (active) {
        int rr = r0 + rl;
        // 4 rows in flight per thread
        for (; rr + 3 * RL < r1; rr += 4 * RL) {
            uint4 v[4];
            float uu[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int row = rr + q * RL;
                int64_t src = row;
                if (GATHER) { src = idx[row]; if (src < 0 || src >= m) src = -1; }
                uu[q] = (src < 0) ? 0.f : u[row];
                v[q] = (src < 0) ? make_uint4(0, 0, 0, 0)
                                 : *reinterpret_cast<const uint4 *>(base + src * ld + (int64_t)cv * kVec);
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) VecTraits<T>::fma_into(acc, v[q], uu[q]);
        }
        for (; rr < r1; rr += RL) {
            int64_t src = rr;
            if (GATHER) { src = idx[rr]; if (src < 0 || src >= m) src = -1; }
            if (src >= 0) {
                const uint4 v = *reinterpret_cast<const uint4 *>(base + src * ld + (int64_t)cv * kVec);
                VecTraits<T>::fma_into(acc, v, u[rr]);
            }
        }
    }
    // reduce over row lanes: red[rl][cvl*kVec + k]
    const int tile_cols = CV * kVec;
#pragma unroll
    for (int k = 0; k < kVec; ++k) red[rl * tile_cols + cvl * kVec + k] = acc[k];
    __syncthreads();
    const int col0 = blockIdx.x * tile_cols;
    if (tid < tile_cols) {
        float sum = 0.f;
        for (int q = 0; q < RL; ++q) sum += red[q * tile_cols + tid];
        if (col0 + tid < n) partial[(int64_t)blockIdx.y * ldp + col0 + tid] = sum;
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = (atomicAdd(&counters[blockIdx.x], 1u) == gridDim.y - 1);
    __syncthreads();
    if (!s_last) { stamp_end(stamp); return; }
    __threadfence();
    float *x = ind ? ind->x : x_direct;
    if (tid < tile_cols && col0 + tid < n) {
        const int col = col0 + tid;
        float g = 0.f;
        for (unsigned q = 0; q < gridDim.y; ++q) g += __ldcg(&partial[(int64_t)q * ldp + col]);
        const float xn = fmaf(-alpha, g, x[col]);
        x[col] = xn;
        if (SHADOW) store_shadow(xbf, split_ld, col, xn);
    }
    if (tid == 0) counters[blockIdx.x] = 0u;
    __syncthreads();
    stamp_end(stamp);
}

// ------------------------------------------------------------------ wide rows: streamed through the copy engine ---
// For rows of >= 512 bytes the BF16 path uses gradient_stream_kernel: a CTA of 16 warps takes a slab of rows and a
// segment of 1024 columns; every warp streams its own rows' 2 KB pieces through a private ring of shared-memory
// slots with cp.async.bulk (lane 0 issues; ~100 KB of reads in flight per SM), each lane keeps 32 column sums in
// registers (u broadcast by shuffle), the 16 warps' sums are added through shared memory, one partial per CTA is
// written, and the last CTA of a column segment adds the partials in a fixed order and applies the update.
constexpr int kGsWarps = 16, kGsDepth = 4, kGsSegCols = 1024;
constexpr uint32_t kGsPiece = kGsSegCols * 2;                 // bytes of one row piece
constexpr size_t kGsSmem = (size_t)kGsWarps * kGsDepth * kGsPiece + (size_t)kGsWarps * kGsSegCols * 4;

__global__ void __launch_bounds__(32 * kGsWarps, 1)
gradient_stream_kernel(const uint16_t *Y, int32_t ldy, int32_t n, int32_t sb, int32_t rpw,
                       const float *u, float alpha, float *x_direct,
                       const StepParams *ind, uint16_t *xbf, int32_t split_ld, float *partial,
                       int32_t ldp, unsigned *counters, unsigned long long *stamp)
{
    extern __shared__ __align__(128) unsigned char gs_smem[];
    __shared__ __align__(8) unsigned long long bars[kGsWarps * kGsDepth];
    __shared__ bool s_last;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    pdl_trigger();
    const uint32_t ring = (uint32_t)__cvta_generic_to_shared(gs_smem) + (uint32_t)warp * (kGsDepth * kGsPiece);
    float *red = reinterpret_cast<float *>(gs_smem + (size_t)kGsWarps * kGsDepth * kGsPiece);      // [16][1024]
    const uint32_t bar0 = (uint32_t)__cvta_generic_to_shared(bars) + 8u * (uint32_t)(warp * kGsDepth);
    if (lane == 0) {
#pragma unroll
        for (int d = 0; d < kGsDepth; ++d)
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar0 + 8u * d) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
    pdl_wait();
    stamp_begin(stamp);

    const int col0 = blockIdx.x * kGsSegCols;
    const uint32_t segB = min(kGsPiece, (uint32_t)(ldy - col0) * 2u);       // a multiple of 16 (ldy % 8 == 0)
    const int r0 = min(sb, (blockIdx.y * kGsWarps + warp) * rpw), r1 = min(sb, r0 + rpw);
    const int nrows = r1 - r0;                                              // <= 32
    const float u_mine = lane < nrows ? ld_dep(u + r0 + lane) : 0.f;
    const uint16_t *src = Y + (int64_t)r0 * ldy + col0;
    // the update is the last reader of the step's rows: they may leave L2 first
    unsigned long long pol_first;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_first));
    auto issue = [&](int k) {
        if (k < nrows && lane == 0) {
            const uint32_t bar = bar0 + 8u * (k % kGsDepth);
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(segB) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                         ::"r"(ring + (uint32_t)(k % kGsDepth) * kGsPiece), "l"(src + (int64_t)k * ldy), "r"(segB), "r"(bar), "l"(pol_first) : "memory");
        }
    };
#pragma unroll 1
    for (int k = 0; k < kGsDepth - 1; ++k) issue(k);
    float acc[4][8];
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int e = 0; e < 8; ++e) acc[c][e] = 0.f;
#pragma unroll 1
    for (int k = 0; k < nrows; ++k) {
        issue(k + kGsDepth - 1);                        // into the slot consumed in the previous iteration
        const float uu = __shfl_sync(0xffffffffu, u_mine, k);
        const uint32_t bar = bar0 + 8u * (k % kGsDepth), parity = (uint32_t)(k / kGsDepth) & 1u;
        uint32_t done;
        do {
            asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                         : "=r"(done) : "r"(bar), "r"(parity) : "memory");
        } while (!done);
        const uint32_t sbase = ring + (uint32_t)(k % kGsDepth) * kGsPiece + (uint32_t)lane * 16u;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            if ((uint32_t)(lane + 32 * c) * 16u < segB) {
                uint4 v;
                asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(sbase + 512u * c));
                VecTraits<uint16_t>::fma_into(acc[c], v, uu);
            }
        }
        __syncwarp();                                   // every lane is done with the slot before it is refilled
    }
    // add the 16 warps' column sums: red[warp][col], col = (lane + 32 c) * 8 + e
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        float4 *dst = reinterpret_cast<float4 *>(red + warp * kGsSegCols + (lane + 32 * c) * 8);
        dst[0] = make_float4(acc[c][0], acc[c][1], acc[c][2], acc[c][3]);
        dst[1] = make_float4(acc[c][4], acc[c][5], acc[c][6], acc[c][7]);
    }
    __syncthreads();
    const int cl = threadIdx.x * 2;                     // this thread's two columns of the segment
    const bool mine = col0 + cl < ldy;
    if (mine) {
        float sx = 0.f, sy = 0.f;
#pragma unroll
        for (int w = 0; w < kGsWarps; ++w) {
            const float2 v = *reinterpret_cast<const float2 *>(red + w * kGsSegCols + cl);
            sx += v.x;
            sy += v.y;
        }
        *reinterpret_cast<float2 *>(partial + (int64_t)blockIdx.y * ldp + col0 + cl) = make_float2(sx, sy);
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(&counters[blockIdx.x], 1u) == gridDim.y - 1);
    __syncthreads();
    if (!s_last) { stamp_end(stamp); return; }
    __threadfence();
    float *x = ind ? ind->x : x_direct;
    if (mine) {
        float gx = 0.f, gy = 0.f;
        // (all loads of a batch of 16 in flight before the first add: the tail is a chain of L2 round trips otherwise)
#pragma unroll 16
        for (unsigned q = 0; q < gridDim.y; ++q) {
            const float2 v = __ldcg(reinterpret_cast<const float2 *>(partial + (int64_t)q * ldp + col0 + cl));
            gx += v.x;
            gy += v.y;
        }
        const int col = col0 + cl;
        if (col < n) {
            const float xn = fmaf(-alpha, gx, x[col]);
            x[col] = xn;
            store_shadow(xbf, split_ld, col, xn);
        }
        if (col + 1 < n) {
            const float xn = fmaf(-alpha, gy, x[col + 1]);
            x[col + 1] = xn;
            store_shadow(xbf, split_ld, col + 1, xn);
        }
    }
    if (threadIdx.x == 0) counters[blockIdx.x] = 0u;
    __syncthreads();
    stamp_end(stamp);
}

cudaError_t gradient_configure()
{
    return cudaFuncSetAttribute(gradient_stream_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kGsSmem);
}

static int launch_gradient_stream(cudaStream_t st, const uint16_t *Y, int32_t ldy, int32_t n, int32_t sb, const float *u,
                                  float alpha, float *x, const StepParams *ind, uint16_t *xbf, const GradWorkspace &ws)
{
    const int col_segs = (ldy + kGsSegCols - 1) / kGsSegCols;
    // rows per warp: at most 32 (one u per lane), at least 2; about one CTA per SM (measured on n = 2000, s*b = 2048:
    // a floor of 8 rows left 32 CTAs for 148 SMs, 7.4 us for 8 MB)
    const int slabs_target = std::max(1, ws.num_sms / col_segs);
    int rpw = (sb + kGsWarps * slabs_target - 1) / (kGsWarps * slabs_target);
    rpw = std::min(32, std::max(2, rpw));
    const int slabs = (sb + kGsWarps * rpw - 1) / (kGsWarps * rpw);
    if (slabs > ws.max_splits) return 0;
    launch_pdl(gradient_stream_kernel, dim3(col_segs, slabs), dim3(32 * kGsWarps), kGsSmem, st, 1, Y, ldy, n, sb, rpw, u, alpha, x,
               ind, xbf, ws.split_ld, ws.partial, ws.ldp, ws.counters, g_stamp);
    return 1;
}

static inline int next_pow2(int v) { int p = 1; while (p < v) p <<= 1; return p; }

template <typename T, bool GATHER, bool SHADOW>
static int launch_gradient_any(cudaStream_t st, const T *base, int64_t ld, const int32_t *idx, int64_t m, int32_t n,
                               int32_t rows, const float *u, float alpha, float *x, const StepParams *ind,
                               uint16_t *xbf, const GradWorkspace &ws)
{
    constexpr int kVec = VecTraits<T>::kVec;
    const int nvec = (n + kVec - 1) / kVec;
    const int CV = min(32, next_pow2(nvec));
    const int RL = kGradThreads / CV;
    const int col_tiles = (nvec + CV - 1) / CV;
    int splits = (4 * ws.num_sms + col_tiles - 1) / col_tiles;
    splits = min(splits, (rows + RL - 1) / RL);
    splits = max(1, min(splits, ws.max_splits));
    const int rows_per_split = (rows + splits - 1) / splits;
    splits = (rows + rows_per_split - 1) / rows_per_split;
    dim3 grid(col_tiles, splits);
    launch_pdl(gradient_update_kernel<T, GATHER, SHADOW>, grid, dim3(kGradThreads), 0, st, 1, base, ld, idx, m, n, rows,
               rows_per_split, CV, u, alpha, x, ind, xbf, ws.split_ld, ws.partial, ws.ldp, ws.counters, SHADOW ? g_stamp : nullptr);
    return 1;
}

int launch_gradient_bf16(cudaStream_t st, const uint16_t *Y, int32_t ldy, int32_t n, int32_t sb, const float *u,
                         float alpha, float *x, const StepParams *ind, uint16_t *xbf, const GradWorkspace &ws)
{
    if (ldy * 2 >= 512 && launch_gradient_stream(st, Y, ldy, n, sb, u, alpha, x, ind, xbf, ws)) return 1;
    return launch_gradient_any<uint16_t, false, true>(st, Y, ldy, nullptr, 0, n, sb, u, alpha, x, ind, xbf, ws);
}

// ------------------------------------------------------------- margin as its own kernel ---
// r = Y x_bf (Alg. 1 line 3; BF16 inputs, FP32 accumulation and output, L231) for the pipelined
// schedule, where the Gram of step t + 1 is computed beside the recurrence of step t, before x(t+1) exists, so that the
// margin can no longer ride in the Gram's B operand. A warp per row, two rows and eight 16-byte loads in flight per
// lane; Y's pad columns and the shadow buffer's are zero, so whole 16-byte vectors are summed.
constexpr int kMgWarps = 16;

__device__ __forceinline__ uint4 ld_stream_v4(const void *p)
{
    uint4 r;
    asm volatile("ld.global.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p) : "memory");
    return r;
}


__global__ void __launch_bounds__(32 * kMgWarps)
margin_kernel(const uint16_t *Y, int32_t ldy, int32_t sb, const uint16_t *xbf, const float *x32, const StepParams *ind,
              int exact, float *r, unsigned long long *stamp)
{
    pdl_trigger();
    pdl_wait();                                     // x_bf comes from the previous update, Y from the gather
    stamp_begin(stamp);
    if (exact) {
        // CASGD_OPT_MARGIN_SPLIT: the margin of the FP32 master (Recipe B's u_r = f, Table 3): r = Y x.
        // Columns beyond n are zero in Y; x has exactly n entries, so the last vector of a row is guarded.
        const float *xs = ind ? ind->x : x32;
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        const int gw = blockIdx.x * kMgWarps + warp, W = gridDim.x * kMgWarps;
        const int nvec = ldy >> 3, n = exact;       // (exact carries n)
        for (int row = gw; row < sb; row += W) {
            const uint16_t *yr = Y + (int64_t)row * ldy;
            float acc = 0.f;
            for (int cv0 = lane; cv0 < nvec; cv0 += 128) {
                uint4 v[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const int cv = cv0 + 32 * q;
                    v[q] = make_uint4(0u, 0u, 0u, 0u);
                    if (cv < nvec) v[q] = ld_stream_v4(yr + cv * 8);
                }
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const int col = (cv0 + 32 * q) * 8;
                    if (col >= n) continue;
                    float xv[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) xv[e] = col + e < n ? ld_dep(xs + col + e) : 0.f;
                    acc = fmaf(bf16lo(v[q].x), xv[0], acc); acc = fmaf(bf16hi(v[q].x), xv[1], acc);
                    acc = fmaf(bf16lo(v[q].y), xv[2], acc); acc = fmaf(bf16hi(v[q].y), xv[3], acc);
                    acc = fmaf(bf16lo(v[q].z), xv[4], acc); acc = fmaf(bf16hi(v[q].z), xv[5], acc);
                    acc = fmaf(bf16lo(v[q].w), xv[6], acc); acc = fmaf(bf16hi(v[q].w), xv[7], acc);
                }
            }
            acc = warp_sum(acc);
            if (lane == 0) r[row] = acc;
        }
        stamp_end_warp(stamp);
        return;
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int gw = blockIdx.x * kMgWarps + warp, W = gridDim.x * kMgWarps;
    const int nvec = ldy >> 3;
    for (int row = 2 * gw; row < sb; row += 2 * W) {
        const bool two = row + 1 < sb;
        const uint16_t *y0 = Y + (int64_t)row * ldy, *y1 = y0 + (two ? ldy : 0);
        float a0 = 0.f, a1 = 0.f;
        for (int cv0 = lane; cv0 < nvec; cv0 += 128) {
            uint4 v0[4], v1[4], xv[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int cv = cv0 + 32 * q;
                v0[q] = v1[q] = make_uint4(0u, 0u, 0u, 0u);
                if (cv < nvec) { v0[q] = ld_stream_v4(y0 + cv * 8); v1[q] = ld_stream_v4(y1 + cv * 8); }
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int cv = cv0 + 32 * q;
                xv[q] = make_uint4(0u, 0u, 0u, 0u);
                if (cv < nvec) xv[q] = ld_dep_v4(xbf + cv * 8);
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) { a0 = dot8_bf16(v0[q], xv[q], a0); a1 = dot8_bf16(v1[q], xv[q], a1); }
        }
        a0 = warp_sum(a0);
        a1 = warp_sum(a1);
        if (lane == 0) { r[row] = a0; if (two) r[row + 1] = a1; }
    }
    stamp_end_warp(stamp);
}

int launch_margin(cudaStream_t st, const uint16_t *Y, int32_t ldy, int32_t n, int32_t sb, const uint16_t *xbf, const float *x32,
                  const StepParams *ind, bool exact, float *r, int num_sms)
{
    const int pairs = (sb + 1) / 2;
    // two CTAs per SM at most: 32 warps x 2 rows x 4 x 16-byte loads per lane = 128 KB in flight per SM
    const int blocks = std::max(1, std::min(2 * num_sms, (pairs + kMgWarps - 1) / kMgWarps));
    launch_pdl(margin_kernel, dim3(blocks), dim3(32 * kMgWarps), 0, st, 1, Y, ldy, sb, xbf, x32, ind, exact ? n : 0, r, g_stamp);
    return 1;
}

// ------------------------------------------------------------- s = 1 with BF16 rows ---
// At s = 1 there is no Gram matrix and no correction: the step is plain mini-batch SGD on BF16 rows with a BF16
// shadow of x (Alg. 1 with s = 1, L99). One warp per sampled row gathers the row from A (16-byte loads), writes it
// to the Y stage (the gradient's second pass and casgd_debug_export read it), forms r = y_i . x_bf in FP32 and
// applies l': gather + margin + residual in one kernel instead of three.
__global__ void __launch_bounds__(256)
margin_s1_kernel(const uint16_t *__restrict__ A, int64_t lda, const float *__restrict__ y, int64_t m, int32_t n,
                 const int32_t *idx, const StepParams *ind, int64_t idx_off, int32_t b, int loss, const uint16_t *xbf,
                 int32_t split_ld, uint16_t *Y, int32_t ldy, float *yI, float *r, float *z, float *u, int *err_flag,
                 unsigned long long *stamp)
{
    pdl_trigger();
    pdl_wait();                                     // x_bf comes from the previous gradient; Y is read by it until now
    stamp_begin(stamp);
    const int row = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (row >= b) return;
    const int32_t *I = ind ? ind->idx + idx_off : idx;
    int64_t src = I[row];
    const bool ok = src >= 0 && src < m;
    float acc = 0.f;
    const int nvec = ldy >> 3;
    for (int cv0 = lane; cv0 < nvec; cv0 += 128) {   // four 16-byte loads of the row in flight per lane
        uint4 v[4], xv[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int col = (cv0 + 32 * q) * 8;
            v[q] = make_uint4(0u, 0u, 0u, 0u);
            if (ok && col < n) v[q] = ldg_nc_v4(A + src * lda + col);
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int col = (cv0 + 32 * q) * 8;
            xv[q] = make_uint4(0u, 0u, 0u, 0u);
            if (col < ldy) xv[q] = ld_dep_v4(xbf + col);     // the shadow buffer is padded to 64 columns with zeros
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int col = (cv0 + 32 * q) * 8;
            if (col >= ldy) continue;
            const int valid = n - col;
            if (valid < 8) {                         // the last chunk of the row: pad columns of Y are zero
                uint32_t w[4] = {v[q].x, v[q].y, v[q].z, v[q].w};
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    if (2 * e >= valid) w[e] = 0u;
                    else if (2 * e + 1 >= valid) w[e] &= 0x0000ffffu;
                }
                v[q] = make_uint4(w[0], w[1], w[2], w[3]);
            }
            *reinterpret_cast<uint4 *>(Y + (int64_t)row * ldy + col) = v[q];
            acc = fmaf(bf16lo(v[q].x), bf16lo(xv[q].x), acc); acc = fmaf(bf16hi(v[q].x), bf16hi(xv[q].x), acc);
            acc = fmaf(bf16lo(v[q].y), bf16lo(xv[q].y), acc); acc = fmaf(bf16hi(v[q].y), bf16hi(xv[q].y), acc);
            acc = fmaf(bf16lo(v[q].z), bf16lo(xv[q].z), acc); acc = fmaf(bf16hi(v[q].z), bf16hi(xv[q].z), acc);
            acc = fmaf(bf16lo(v[q].w), bf16lo(xv[q].w), acc); acc = fmaf(bf16hi(v[q].w), bf16hi(xv[q].w), acc);
            if (split_ld) {                          // CASGD_OPT_MARGIN_SPLIT: the residue rows of the shadow
                acc = dot8_bf16(v[q], ld_dep_v4(xbf + split_ld + col), acc);
                acc = dot8_bf16(v[q], ld_dep_v4(xbf + 2 * split_ld + col), acc);
            }
        }
    }
    acc = warp_sum(acc);
    if (lane == 0) {
        const float ylab = ok ? y[src] : 0.f;
        if (!ok) flag_index_error(err_flag);
        yI[row] = ylab;
        r[row] = acc;
        z[row] = acc;
        u[row] = lprime_rt(loss, acc, ylab);
    }
    stamp_end_warp(stamp);
}

int launch_margin_s1(cudaStream_t st, const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n,
                     const int32_t *idx, const StepParams *ind, int64_t idx_off, int32_t b, int loss, const uint16_t *xbf,
                     int32_t split_ld, uint16_t *Y, int32_t ldy, float *yI, float *r, float *z, float *u, int *err_flag)
{
    launch_pdl(margin_s1_kernel, dim3((b * 32 + 255) / 256), dim3(256), 0, st, 1, A, lda, y, m, n, idx, ind, idx_off, b, loss, xbf,
               split_ld, Y, ldy, yI, r, z, u, err_flag, g_stamp);
    return 1;
}

// ------------------------------------------------------------- FP32 s = 1 baseline ---

// z_i = a32_{I_i}^T x ; u_i = l'(z_i, y_{I_i}); one warp per row, everything FP32.
__global__ void __launch_bounds__(256)
sgd32_margin_kernel(const float *__restrict__ A32, int64_t lda32, const float *__restrict__ y, int64_t m, int32_t n,
                    const int32_t *idx, int32_t b, int loss, const float *x, float *z,
                    float *u, int *err_flag)
{
    pdl_trigger();
    pdl_wait();
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (warp >= b) return;
    const int64_t src = idx[warp];
    if (src < 0 || src >= m) {
        if (lane == 0) { z[warp] = 0.f; u[warp] = 0.f; flag_index_error(err_flag); }
        return;
    }
    const float *a = A32 + src * lda32;
    float acc = 0.f;
    const int n4 = n & ~3;
    for (int k = lane * 4; k < n4; k += 128) {
        const float4 av = *reinterpret_cast<const float4 *>(a + k);
        const float4 xv = *reinterpret_cast<const float4 *>(x + k);
        acc = fmaf(av.x, xv.x, acc); acc = fmaf(av.y, xv.y, acc);
        acc = fmaf(av.z, xv.z, acc); acc = fmaf(av.w, xv.w, acc);
    }
    for (int k = n4 + lane; k < n; k += 32) acc = fmaf(a[k], x[k], acc);
    acc = warp_sum(acc);
    if (lane == 0) {
        z[warp] = acc;
        u[warp] = lprime_rt(loss, acc, y[src]);
    }
}

int launch_sgd32_step(cudaStream_t st, const float *A32, int64_t lda32, const float *y, int64_t m, int32_t n,
                      const int32_t *idx, int32_t b, float alpha, int loss, float *x, float *u, float *z,
                      int *err_flag, const GradWorkspace &ws)
{
    launch_pdl(sgd32_margin_kernel, dim3((b * 32 + 255) / 256), dim3(256), 0, st, 1, A32, lda32, y, m, n, idx, b, loss,
               (const float *)x, z, u, err_flag);
    launch_gradient_any<float, true, false>(st, A32, lda32, idx, m, n, b, u, alpha, x, nullptr, nullptr, ws);
    return 2;
}

}  // namespace casgd

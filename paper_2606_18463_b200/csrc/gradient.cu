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
gradient_update_kernel(const T *__restrict__ base, int64_t ld, const int32_t *__restrict__ idx, int64_t m, int32_t n,
                       int32_t rows, int32_t rows_per_split, int32_t CV, const float *__restrict__ u, float alpha,
                       float *__restrict__ x_direct, const StepParams *__restrict__ ind, uint16_t *__restrict__ xbf,
                       float *__restrict__ partial, int32_t ldp, unsigned *__restrict__ counters)
{
    constexpr int kVec = VecTraits<T>::kVec;
    pdl_trigger();
    pdl_wait();
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
    if (!s_last) return;
    __threadfence();
    float *x = ind ? ind->x : x_direct;
    if (tid < tile_cols && col0 + tid < n) {
        const int col = col0 + tid;
        float g = 0.f;
        for (unsigned q = 0; q < gridDim.y; ++q) g += __ldcg(&partial[(int64_t)q * ldp + col]);
        const float xn = fmaf(-alpha, g, x[col]);
        x[col] = xn;
        if (SHADOW) xbf[col] = f32_to_bf16_bits_rn(xn);
    }
    if (tid == 0) counters[blockIdx.x] = 0u;
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
    int splits = (4 * kNumSMsB200 + col_tiles - 1) / col_tiles;
    splits = min(splits, (rows + RL - 1) / RL);
    splits = max(1, min(splits, ws.max_splits));
    const int rows_per_split = (rows + splits - 1) / splits;
    splits = (rows + rows_per_split - 1) / rows_per_split;
    dim3 grid(col_tiles, splits);
    launch_pdl(gradient_update_kernel<T, GATHER, SHADOW>, grid, dim3(kGradThreads), 0, st, 1, base, ld, idx, m, n, rows,
               rows_per_split, CV, u, alpha, x, ind, xbf, ws.partial, ws.ldp, ws.counters);
    return 1;
}

int launch_gradient_bf16(cudaStream_t st, const uint16_t *Y, int32_t ldy, int32_t n, int32_t sb, const float *u,
                         float alpha, float *x, const StepParams *ind, uint16_t *xbf, const GradWorkspace &ws)
{
    return launch_gradient_any<uint16_t, false, true>(st, Y, ldy, nullptr, 0, n, sb, u, alpha, x, ind, xbf, ws);
}

// ------------------------------------------------------------- FP32 s = 1 baseline ---

// z_i = a32_{I_i}^T x ; u_i = l'(z_i, y_{I_i}); one warp per row, everything FP32.
__global__ void __launch_bounds__(256)
sgd32_margin_kernel(const float *__restrict__ A32, int64_t lda32, const float *__restrict__ y, int64_t m, int32_t n,
                    const int32_t *__restrict__ idx, int32_t b, int loss, const float *__restrict__ x, float *__restrict__ z,
                    float *__restrict__ u, int *__restrict__ err_flag)
{
    pdl_trigger();
    pdl_wait();
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (warp >= b) return;
    const int64_t src = idx[warp];
    if (src < 0 || src >= m) {
        if (lane == 0) { z[warp] = 0.f; u[warp] = 0.f; atomicOr(err_flag, 1); }
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

// loss.cu -- F(x) = (1/m) sum_i L(a_i^T x, y_i): one streaming pass over the BF16 matrix A.
// A pure HBM-bound GEMV (2 m n bytes): 16-byte read-only loads that bypass L1, x staged once per CTA
// in shared memory as FP32, FP32 margins and per-row losses, FP64 accumulation, deterministic
// two-kernel reduction (per-CTA partials, then one CTA sums them in order).
#include <algorithm>

#include "common.cuh"

namespace casgd {

constexpr int kLossThreads = 512;

// GS lanes cooperate on one row (GS = 32: a warp per row; smaller for narrow rows such as n = 18).
template <int GS>
__global__ void __launch_bounds__(kLossThreads)
loss_rows_kernel(const uint16_t *__restrict__ A, int64_t lda, const float *__restrict__ y, int64_t m, int32_t n,
                 int loss, const float *__restrict__ x, int x_in_smem, double *__restrict__ block_partials)
{
    extern __shared__ __align__(16) float xs[];       // [round_up(n, 8)] when x_in_smem
    __shared__ double warp_part[kLossThreads / 32];
    const int nvec = (n + 7) >> 3;
    if (x_in_smem) {
        for (int k = threadIdx.x; k < nvec * 8; k += blockDim.x) xs[k] = (k < n) ? x[k] : 0.f;
        __syncthreads();
    }
    const float *xv = x_in_smem ? xs : x;
    const int lane_in_group = threadIdx.x % GS;
    const int64_t group = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / GS;
    const int64_t ngroups = (int64_t)gridDim.x * blockDim.x / GS;
    double local = 0.0;
    const int64_t passes = (m + ngroups - 1) / ngroups;      // same trip count for every lane of a warp
    for (int64_t pass = 0; pass < passes; ++pass) {
        const int64_t row = group + pass * ngroups;
        const bool valid = row < m;
        float acc0 = 0.f, acc1 = 0.f;
        if (valid) {
            const uint16_t *a = A + row * lda;
            int c = lane_in_group;
            for (; c + GS < nvec; c += 2 * GS) {           // two 16-byte loads in flight per lane
                const uint4 v0 = ldg_nc_v4(a + c * 8);
                const uint4 v1 = ldg_nc_v4(a + (c + GS) * 8);
                const float4 *p0 = reinterpret_cast<const float4 *>(xv + c * 8);
                const float4 *p1 = reinterpret_cast<const float4 *>(xv + (c + GS) * 8);
                acc0 = dot8(v0, p0[0], p0[1], acc0);
                acc1 = dot8(v1, p1[0], p1[1], acc1);
            }
            if (c < nvec) {
                const uint4 v = ldg_nc_v4(a + c * 8);
                if (!x_in_smem && c * 8 + 8 > n) {         // global x has no zero padding: mask the tail
                    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
                    for (int q = 0; q < 8 && c * 8 + q < n; ++q)
                        acc0 = fmaf((q & 1) ? bf16hi(w[q >> 1]) : bf16lo(w[q >> 1]), x[c * 8 + q], acc0);
                } else {
                    const float4 *p = reinterpret_cast<const float4 *>(xv + c * 8);
                    acc0 = dot8(v, p[0], p[1], acc0);
                }
            }
        }
        float acc = acc0 + acc1;
#pragma unroll
        for (int o = GS / 2; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (valid && lane_in_group == 0) local += (double)loss_value_rt(loss, acc, y[row]);
    }
    local = warp_sum(local);
    if ((threadIdx.x & 31) == 0) warp_part[threadIdx.x >> 5] = local;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int w = 0; w < kLossThreads / 32; ++w) tot += warp_part[w];
        block_partials[blockIdx.x] = tot;
    }
}

__global__ void loss_finish_kernel(const double *__restrict__ block_partials, int32_t nblocks, int64_t m,
                                   double *__restrict__ result)
{
    __shared__ double part[32];
    double v = 0.0;
    for (int i = threadIdx.x; i < nblocks; i += blockDim.x) v += block_partials[i];
    v = warp_sum(v);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) tot += part[w];
        *result = tot / (double)m;
    }
}

int launch_loss(cudaStream_t st, const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n, int loss,
                const float *x, double *block_partials, int32_t max_blocks, double *result_dev)
{
    const int nvec = (n + 7) >> 3;
    const size_t smem_x = sizeof(float) * (size_t)nvec * 8;
    const int x_in_smem = smem_x <= 96 * 1024;
    const size_t smem = x_in_smem ? smem_x : 0;
    // resident CTAs per SM: 2048 threads / 512, or fewer when x fills shared memory
    int per_sm = 4;
    if (smem > 0) per_sm = (int)std::min<size_t>(4, (200 * 1024) / (smem + 1024));
    per_sm = std::max(per_sm, 1);
    int blocks = std::min(max_blocks, kNumSMsB200 * per_sm);
    auto go = [&](auto kern, int gs) {
        int64_t rows_per_pass = (int64_t)blocks * kLossThreads / gs;
        if (rows_per_pass > m) blocks = (int)std::max<int64_t>(1, (m * gs + kLossThreads - 1) / kLossThreads);
        if (smem > 48 * 1024) cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        kern<<<blocks, kLossThreads, smem, st>>>(A, lda, y, m, n, loss, x, x_in_smem, block_partials);
    };
    if (nvec >= 32) go(loss_rows_kernel<32>, 32);
    else if (nvec > 8) go(loss_rows_kernel<16>, 16);
    else if (nvec > 4) go(loss_rows_kernel<8>, 8);
    else if (nvec > 2) go(loss_rows_kernel<4>, 4);
    else if (nvec > 1) go(loss_rows_kernel<2>, 2);
    else go(loss_rows_kernel<1>, 1);
    loss_finish_kernel<<<1, 256, 0, st>>>(block_partials, blocks, m, result_dev);
    return 2;
}

}  // namespace casgd

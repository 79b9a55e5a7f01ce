// recurrence.cu -- the s-step inner residual correction, Alg. 1 lines 6-15:
//   for j = 0..s-1:  z_j = r_j - alpha * sum_{k<j} G_{jk} u_k ;  u_j = l'(z_j, y_{I_j})
// All FP32 (the paper requires u_c = u_sigma = FP32: L236, Table 3). Only blocks k < j of G are read
// ("strict block-lower", L180). The chain is serial in j; inside a step the b rows and the j*b-long
// dot products are parallel.
#include "common.cuh"

namespace casgd {

// v1: one CTA. G_{j,<j} streams from L2/HBM with 16-byte loads, u lives in shared memory,
// warp-shuffle reductions, the loss's link derivative inlined.
template <int LOSS>
__global__ void __launch_bounds__(1024)
recurrence_cta_kernel(const float *__restrict__ G, int32_t ldg, const float *__restrict__ r, const float *__restrict__ yI,
                      int32_t s, int32_t b, float alpha, float *__restrict__ z, float *__restrict__ u)
{
    extern __shared__ float u_s[];                    // [s*b]
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    for (int j = 0; j < s; ++j) {
        const int len = j * b;
        const int len4 = len & ~3;
        for (int i = warp; i < b; i += nwarps) {
            const int row = j * b + i;
            const float *g = G + (int64_t)row * ldg;
            float acc = 0.f;
            for (int t = lane * 4; t < len4; t += 128) {
                const float4 gv = *reinterpret_cast<const float4 *>(g + t);
                const float4 uv = *reinterpret_cast<const float4 *>(u_s + t);
                acc = fmaf(gv.x, uv.x, acc);
                acc = fmaf(gv.y, uv.y, acc);
                acc = fmaf(gv.z, uv.z, acc);
                acc = fmaf(gv.w, uv.w, acc);
            }
            for (int t = len4 + lane; t < len; t += 32) acc = fmaf(g[t], u_s[t], acc);
            acc = warp_sum(acc);
            if (lane == 0) {
                const float zz = fmaf(-alpha, acc, r[row]);
                const float uu = lprime<LOSS>(zz, yI[row]);
                z[row] = zz;
                u[row] = uu;
                u_s[row] = uu;
            }
        }
        __syncthreads();
    }
}

int launch_recurrence(cudaStream_t st, const float *G, int32_t ldg, const float *r, const float *yI, int32_t s,
                      int32_t b, float alpha, int loss, float *z, float *u)
{
    const size_t smem = sizeof(float) * (size_t)s * b;
    const int threads = (b >= 32) ? 1024 : 32 * ((b < 4) ? 4 : b);
    auto go = [&](auto kern) {
        static bool attr_set = false;
        if (!attr_set) {
            cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, CASGD_MAX_SB * (int)sizeof(float));
            attr_set = true;
        }
        kern<<<1, threads, smem, st>>>(G, ldg, r, yI, s, b, alpha, z, u);
    };
    if (loss == CASGD_LOGISTIC) go(recurrence_cta_kernel<CASGD_LOGISTIC>);
    else if (loss == CASGD_LINEAR) go(recurrence_cta_kernel<CASGD_LINEAR>);
    else go(recurrence_cta_kernel<CASGD_POISSON>);
    return 1;
}

}  // namespace casgd

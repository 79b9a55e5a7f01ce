// gram_simt.cu -- bring-up / cross-check Gram + margin kernel on the FP32 FMA pipes.
// Same arithmetic contract as the tcgen05 kernel (BF16 inputs, exact products, FP32 accumulation),
// Alg. 1 lines 3-4. Selected with CASGD_OPT_GRAM_IMPL = 1; not the fast path.
#include "common.cuh"

namespace casgd {

constexpr int ST = 64;   // SIMT tile edge
constexpr int SK = 32;   // K chunk

// needed(ti, tj): does the 64x64 tile hold any entry of a block strictly below the block diagonal?
__device__ __forceinline__ bool tile_needed(int row0, int col0, int edge, int sb, int b, int full_lower)
{
    if (full_lower) return true;
    int last_row = min(row0 + edge, sb) - 1;
    return (last_row / b) > (col0 / b);
}

__global__ void __launch_bounds__(256)
gram_simt_kernel(const uint16_t *__restrict__ Y, int32_t ldy, int32_t n, int32_t sb, int32_t b, float *__restrict__ G,
                 int32_t ldg, int32_t T, int full_lower)
{
    // lower-triangular tile enumeration: blockIdx.x -> (ti, tj), tj <= ti
    int t = blockIdx.x;
    int ti = (int)floorf((sqrtf(8.f * (float)t + 1.f) - 1.f) * 0.5f);
    while ((ti + 1) * (ti + 2) / 2 <= t) ++ti;
    while (ti * (ti + 1) / 2 > t) --ti;
    int tj = t - ti * (ti + 1) / 2;
    const int row0 = ti * ST, col0 = tj * ST;
    if (!tile_needed(row0, col0, ST, sb, b, full_lower)) return;

    __shared__ float As[SK][ST + 1];
    __shared__ float Bs[SK][ST + 1];
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    float acc[4][4] = {};
    for (int k0 = 0; k0 < n; k0 += SK) {
        for (int e = threadIdx.x; e < ST * SK; e += 256) {
            int rr = e / SK, kk = e % SK;
            int k = k0 + kk;
            int ra = row0 + rr, rb = col0 + rr;
            As[kk][rr] = (ra < sb && k < n) ? bf16_bits_to_f32(Y[(int64_t)ra * ldy + k]) : 0.f;
            Bs[kk][rr] = (rb < sb && k < n) ? bf16_bits_to_f32(Y[(int64_t)rb * ldy + k]) : 0.f;
        }
        __syncthreads();
#pragma unroll 8
        for (int kk = 0; kk < SK; ++kk) {
            float a[4], c[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) { a[q] = As[kk][ty * 4 + q]; c[q] = Bs[kk][tx * 4 + q]; }
#pragma unroll
            for (int p = 0; p < 4; ++p)
#pragma unroll
                for (int q = 0; q < 4; ++q) acc[p][q] = fmaf(a[p], c[q], acc[p][q]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int p = 0; p < 4; ++p) {
        int row = row0 + ty * 4 + p;
        if (row >= sb) continue;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            int col = col0 + tx * 4 + q;
            if (col < sb) G[(int64_t)row * ldg + col] = acc[p][q];
        }
    }
}

// r = Y x_bf, one warp per row, FP32 accumulation.
__global__ void __launch_bounds__(256)
margin_simt_kernel(const uint16_t *__restrict__ Y, int32_t ldy, int32_t n, int32_t sb, const uint16_t *xbf, int32_t split_ld,
                   float *__restrict__ r)
{
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (warp >= sb) return;
    float acc = 0.f;
    for (int k = lane; k < n; k += 32) {
        float xv = bf16_bits_to_f32(xbf[k]);
        if (split_ld) xv += bf16_bits_to_f32(xbf[split_ld + k]) + bf16_bits_to_f32(xbf[2 * split_ld + k]);   // == x, exactly
        acc = fmaf(bf16_bits_to_f32(Y[(int64_t)warp * ldy + k]), xv, acc);
    }
    acc = warp_sum(acc);
    if (lane == 0) r[warp] = acc;
}

int launch_gram_simt(cudaStream_t st, const uint16_t *Y, int32_t ldy, int32_t n, int32_t sb, int32_t b,
                     const uint16_t *xbf, int32_t split_ld, float *G, int32_t ldg, float *r, int full_lower)
{
    const int T = (sb + ST - 1) / ST;
    int launches = 1;
    margin_simt_kernel<<<(sb * 32 + 255) / 256, 256, 0, st>>>(Y, ldy, n, sb, xbf, split_ld, r);
    if (full_lower || sb > b) {
        gram_simt_kernel<<<T * (T + 1) / 2, 256, 0, st>>>(Y, ldy, n, sb, b, G, ldg, T, full_lower);
        ++launches;
    }
    return launches;
}

}  // namespace casgd

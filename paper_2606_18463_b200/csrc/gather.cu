// gather.cu -- Alg. 1 line 2: Y = A[I, :], y_I = y[I]; bit-exact copies.
// Also the one-off layout kernels (repack to a padded row stride, FP32 widening, BF16 shadow).
#include "common.cuh"

namespace casgd {

// One thread per 16-byte chunk (8 BF16) of a gathered row. Rows of A are 16-byte aligned
// (lda % 8 == 0), so each row is read with whole 16-byte vector loads; the last chunk of a row is
// masked to n so that the pad columns [n, ldy) of Y are always zero whatever A's padding holds.
__global__ void __launch_bounds__(256)
gather_rows_kernel(const uint16_t *__restrict__ A, int64_t lda, const float *__restrict__ y, int64_t m, int32_t n,
                   const int32_t *__restrict__ idx, const StepParams *__restrict__ ind, int64_t idx_off, int32_t sb,
                   uint16_t *__restrict__ Y, int32_t ldy, float *__restrict__ yI, int *__restrict__ err_flag)
{
    pdl_trigger();
    pdl_wait();                                     // Y is still being read by the previous step's gradient
    const int32_t chunks = ldy >> 3;
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t row = t / chunks;
    const int32_t c = (int32_t)(t - row * chunks);
    if (row >= sb) return;
    const int32_t *I = ind ? ind->idx + idx_off : idx;
    const int64_t src = I[row];
    const bool ok = (src >= 0) && (src < m);
    uint4 v = make_uint4(0u, 0u, 0u, 0u);
    const int32_t col = c << 3;
    if (ok) {
        v = ldg_nc_v4(A + src * lda + col);
        const int32_t valid = n - col;              // elements of this chunk inside the row
        if (valid < 8) {
            uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                if (2 * q >= valid) w[q] = 0u;
                else if (2 * q + 1 >= valid) w[q] &= 0x0000ffffu;
            }
            v = make_uint4(w[0], w[1], w[2], w[3]);
        }
    }
    *reinterpret_cast<uint4 *>(Y + row * (int64_t)ldy + col) = v;
    if (c == 0) {
        yI[row] = ok ? y[src] : 0.f;
        if (!ok) atomicOr(err_flag, 1);
    }
}

int launch_gather(cudaStream_t st, const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n,
                  const int32_t *idx, const StepParams *ind, int64_t idx_off, int32_t sb, uint16_t *Y, int32_t ldy,
                  float *yI, int *err_flag)
{
    const int64_t total = (int64_t)sb * (ldy >> 3);
    const int threads = 256;
    const unsigned blocks = (unsigned)((total + threads - 1) / threads);
    launch_pdl(gather_rows_kernel, dim3(blocks), dim3(threads), 0, st, 1, A, lda, y, m, n, idx, ind, idx_off, sb, Y, ldy, yI,
               err_flag);
    return 1;
}

// x_bf = bf16_rne(x): the margin kernel's view of the weights.
__global__ void shadow_kernel(const float *__restrict__ x, const StepParams *__restrict__ ind, int32_t n,
                              uint16_t *__restrict__ xbf)
{
    pdl_trigger();
    pdl_wait();
    const float *xs = ind ? ind->x : x;
    int32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) xbf[k] = f32_to_bf16_bits_rn(xs[k]);
}

int launch_shadow(cudaStream_t st, const float *x, const StepParams *ind, int32_t n, uint16_t *xbf)
{
    launch_pdl(shadow_kernel, dim3((n + 255) / 256), dim3(256), 0, st, 1, x, ind, n, xbf);
    return 1;
}

// Exact FP32 widening of A for the all-FP32 baseline (Recipe A storage, Table 3).
__global__ void widen_kernel(const uint16_t *__restrict__ A, int64_t lda, int64_t m, int32_t n, float *__restrict__ A32,
                             int64_t lda32)
{
    const int64_t total = m * lda32;
    for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
        const int64_t row = t / lda32;
        const int32_t k = (int32_t)(t - row * lda32);
        A32[t] = (k < n) ? bf16_bits_to_f32(A[row * lda + k]) : 0.f;
    }
}

int launch_widen(cudaStream_t st, const uint16_t *A, int64_t lda, int64_t m, int32_t n, float *A32, int64_t lda32)
{
    widen_kernel<<<kNumSMsB200 * 8, 256, 0, st>>>(A, lda, m, n, A32, lda32);
    return 1;
}

// Copy X (any row stride) into the library's padded layout; pad columns are zero.
__global__ void repack_kernel(const uint16_t *__restrict__ X, int64_t ldx, int64_t m, int32_t n, uint16_t *__restrict__ A,
                              int64_t lda)
{
    const int64_t total = m * lda;
    for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
        const int64_t row = t / lda;
        const int32_t k = (int32_t)(t - row * lda);
        A[t] = (k < n) ? X[row * ldx + k] : (uint16_t)0;
    }
}

int launch_repack(cudaStream_t st, const uint16_t *X, int64_t ldx, int64_t m, int32_t n, uint16_t *A, int64_t lda)
{
    repack_kernel<<<kNumSMsB200 * 8, 256, 0, st>>>(X, ldx, m, n, A, lda);
    return 1;
}

__global__ void set_params_kernel(StepParams *ind, const int32_t *idx, float *x)
{
    pdl_trigger();
    pdl_wait();                                     // the previous replay may still be reading the block
    ind->idx = idx;
    ind->x = x;
}

int launch_set_params(cudaStream_t st, StepParams *ind, const int32_t *idx, float *x)
{
    launch_pdl(set_params_kernel, dim3(1), dim3(1), 0, st, 1, ind, idx, x);
    return 1;
}

}  // namespace casgd

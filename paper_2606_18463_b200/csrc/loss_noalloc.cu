// loss_noalloc.cu -- casgd_loss_noalloc: F(x) = (1/m) sum_i L(a_i^T x, y_i) for callers that cannot
// allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc. A variant of
// loss_rows_kernel (loss.cu) -- plain loads of the BF16 rows, FP32 margins and per-row losses, FP64 sums -- whose scratch
// (the partial sums that loss.cu keeps in a context's cudaMalloc'ed block_partials) lives in ONE file-scope
// `static __device__` array: no context, no cudaMalloc / cudaFree / allocating library call, inputs and output the caller's.
//
// Scratch: kNaMaxChunks doubles = 128 KB, held by every GPU that loads the library until the process exits. One double
// per chunk of kNaChunkRows = 256 rows, so m <= 256 * 16384 = 4,194,304 rows; larger m is rejected (CASGD_EINVAL).
// Every chunk's slot is WRITTEN before the finishing kernel reads it, so nothing has to start at zero and the last
// call's contents do not matter. All calls on a device share the array: calls that OVERLAP on the GPU (different
// streams, or graphs replayed concurrently) race; calls on one stream are ordered and safe.
// The summation order is fixed by (m, n) alone -- rows of a chunk in order, chunks in order -- whatever the grid.
#include <algorithm>
#include <cstdio>
#include <mutex>

#include "common.cuh"

namespace casgd {

namespace {

constexpr int kNaChunkRows = 256, kNaMaxChunks = 16384, kNaThreads = 256, kNaWarps = 8;
constexpr int kNaMaxDevices = 64;

static __device__ __align__(256) double g_loss_noalloc_scratch[kNaMaxChunks];

// In host code the array's name is a host-side stand-in, not a device address: the kernels get the address that
// cudaGetSymbolAddress returns for the CURRENT device, resolved once per device (set-up; not an allocation).
std::mutex g_na_mutex;
double *g_na_scratch_of[kNaMaxDevices];
thread_local char g_na_error[256];

// VEC: rows are 16-byte aligned (X and ldx): 16-byte loads, 8 columns per lane and pass; else 2-byte loads.
template <bool VEC>
__global__ void __launch_bounds__(kNaThreads)
loss_noalloc_kernel(const uint16_t *X, int64_t ldx, const float *y, int64_t m, int32_t n, int loss, const float *x,
                    double *scratch, int32_t nchunks)
{
    __shared__ double warp_part[kNaWarps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int32_t chunk = blockIdx.x; chunk < nchunks; chunk += gridDim.x) {
        const int64_t row0 = (int64_t)chunk * kNaChunkRows + warp * (kNaChunkRows / kNaWarps);
        double local = 0.0;                              // lane 0: this warp's 32 rows, in row order
        for (int k = 0; k < kNaChunkRows / kNaWarps; ++k) {
            const int64_t row = row0 + k;
            if (row >= m) break;                         // (uniform over the warp)
            const uint16_t *a = X + row * ldx;
            float acc = 0.f;
            if (VEC) {
                const int nvec = n >> 3;
                for (int c = lane; c < nvec; c += 32) {
                    const uint4 v = ldg_nc_v4(a + c * 8);
                    const float *xv = x + c * 8;
                    acc = fmaf(bf16lo(v.x), xv[0], acc); acc = fmaf(bf16hi(v.x), xv[1], acc);
                    acc = fmaf(bf16lo(v.y), xv[2], acc); acc = fmaf(bf16hi(v.y), xv[3], acc);
                    acc = fmaf(bf16lo(v.z), xv[4], acc); acc = fmaf(bf16hi(v.z), xv[5], acc);
                    acc = fmaf(bf16lo(v.w), xv[6], acc); acc = fmaf(bf16hi(v.w), xv[7], acc);
                }
                for (int c = nvec * 8 + lane; c < n; c += 32) acc = fmaf(__uint_as_float((uint32_t)a[c] << 16), x[c], acc);
            } else {
                for (int c = lane; c < n; c += 32) acc = fmaf(__uint_as_float((uint32_t)a[c] << 16), x[c], acc);
            }
            acc = warp_sum(acc);
            if (lane == 0) local += (double)loss_value_rt(loss, acc, y[row]);
        }
        if (lane == 0) warp_part[warp] = local;
        __syncthreads();
        if (threadIdx.x == 0) {
            double tot = 0.0;
            for (int w = 0; w < kNaWarps; ++w) tot += warp_part[w];
            scratch[chunk] = tot;
        }
        __syncthreads();
    }
}

__global__ void __launch_bounds__(kNaThreads)
loss_noalloc_finish_kernel(const double *scratch, int32_t nchunks, int64_t m, double *result)
{
    __shared__ double part[kNaThreads];
    double v = 0.0;
    for (int i = threadIdx.x; i < nchunks; i += kNaThreads) v += scratch[i];
    part[threadIdx.x] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int t = 0; t < kNaThreads; ++t) tot += part[t];
        *result = tot / (double)m;
    }
}

int na_fail(int code, const char *msg)
{
    snprintf(g_na_error, sizeof g_na_error, "%s", msg);
    return code;
}

}  // namespace

}  // namespace casgd

using namespace casgd;

extern "C" {

const char *casgd_loss_noalloc_error(void) { return g_na_error; }

int casgd_loss_noalloc(const uint16_t *X_bf16, int64_t ldx, const float *y, int64_t m, int32_t n, int loss, const float *x,
                       double *result_dev, void *cuda_stream)
{
    g_na_error[0] = 0;
    if (!X_bf16 || !y || !x || !result_dev) return na_fail(CASGD_EINVAL, "casgd_loss_noalloc: null pointer");
    if (m < 1 || n < 1 || ldx < n || loss < 0 || loss > 2) return na_fail(CASGD_EINVAL, "casgd_loss_noalloc: bad m, n, ldx or loss");
    if (m > (int64_t)kNaChunkRows * kNaMaxChunks) {
        snprintf(g_na_error, sizeof g_na_error,
                 "casgd_loss_noalloc: m = %lld exceeds the static scratch (at most %lld rows: %d partial sums of %d rows)",
                 (long long)m, (long long)kNaChunkRows * kNaMaxChunks, kNaMaxChunks, kNaChunkRows);
        return CASGD_EINVAL;
    }
    int dev = -1;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kNaMaxDevices)
        return na_fail(CASGD_ECUDA, "casgd_loss_noalloc: no current device (or its ordinal is beyond 63)");
    double *scratch = nullptr;
    int sms = 0;
    {
        std::lock_guard<std::mutex> lock(g_na_mutex);
        if (!g_na_scratch_of[dev]) {                     // set-up, once per device, with that device current
            if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return na_fail(CASGD_ECUDA, "casgd_loss_noalloc: cudaGetDeviceProperties failed");
            if (prop.major != 10) return na_fail(CASGD_EARCH, "casgd_loss_noalloc: the current device is not sm_100");
            void *p = nullptr;
            const cudaError_t e = cudaGetSymbolAddress(&p, g_loss_noalloc_scratch);
            if (e != cudaSuccess || !p) {
                snprintf(g_na_error, sizeof g_na_error, "casgd_loss_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
                return CASGD_ECUDA;
            }
            g_na_scratch_of[dev] = static_cast<double *>(p);
        }
        scratch = g_na_scratch_of[dev];
    }
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) sms = 148;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int32_t nchunks = (int32_t)((m + kNaChunkRows - 1) / kNaChunkRows);
    const int blocks = std::min<int32_t>(nchunks, 8 * sms);
    const bool vec = ((uintptr_t)X_bf16 % 16 == 0) && (ldx % 8 == 0) && ((uintptr_t)x % 4 == 0);
    if (vec) loss_noalloc_kernel<true><<<blocks, kNaThreads, 0, st>>>(X_bf16, ldx, y, m, n, loss, x, scratch, nchunks);
    else loss_noalloc_kernel<false><<<blocks, kNaThreads, 0, st>>>(X_bf16, ldx, y, m, n, loss, x, scratch, nchunks);
    loss_noalloc_finish_kernel<<<1, kNaThreads, 0, st>>>(scratch, nchunks, m, result_dev);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(g_na_error, sizeof g_na_error, "casgd_loss_noalloc: launch: %s", cudaGetErrorString(e));
        return CASGD_ECUDA;
    }
    return CASGD_OK;
}

}  // extern "C"

// gather.cu -- Alg. 1 line 2: Y = A[I, :], y_I = y[I]; bit-exact copies.
// Also the one-off layout kernels (repack to a padded row stride, FP32 widening, BF16 shadow).
#include "common.cuh"

namespace casgd {

// One thread per 16-byte chunk (8 BF16) of a gathered row. Rows of A are 16-byte aligned
// (lda % 8 == 0), so each row is read with whole 16-byte vector loads; the last chunk of a row is
// masked to n so that the pad columns [n, ldy) of Y are always zero whatever A's padding holds.
__global__ void __launch_bounds__(256)
gather_rows_kernel(const uint16_t *__restrict__ A, int64_t lda, const float *__restrict__ y, int64_t m, int32_t n,
                   const int32_t *idx, const StepParams *ind, int64_t idx_off, int32_t sb,
                   uint16_t *Y, int32_t ldy, float *yI, int *err_flag, unsigned long long *stamp)
{
    pdl_trigger();
    pdl_wait();                                     // Y is still being read by the previous step's gradient
    stamp_begin(stamp);
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
        if (!ok) flag_index_error(err_flag);
    }
    stamp_end_warp(stamp);
}

// Wide rows (n % 8 == 0, >= 512 bytes): the gather is pure data movement, so it is done by the copy engine alone.
// One lane per warp drives a ring of kGbDepth 4 KB shared-memory slots (kGbAhead loads in flight): cp.async.bulk global -> shared for a piece
// of a sampled row, then cp.async.bulk shared -> global into the Y stage; no byte passes through a register, and
// each SM keeps ~100 KB of reads in flight. The row indices of a warp's next 32 rows are loaded by its 32 lanes
// at once. Labels and the out-of-range check are done by the first warps of the grid, element-wise.
constexpr int kGbWarps = 8, kGbDepth = 6, kGbAhead = 4;
constexpr uint32_t kGbSlot = 4096;

__global__ void __launch_bounds__(32 * kGbWarps, 1)
gather_bulk_kernel(const uint16_t *__restrict__ A, int64_t lda, const float *__restrict__ y, int64_t m, int32_t n,
                   const int32_t *idx, const StepParams *ind, int64_t idx_off, int32_t sb,
                   uint16_t *Y, int32_t ldy, float *yI, int *err_flag, unsigned long long *stamp)
{
    extern __shared__ __align__(128) unsigned char gb_smem[];
    __shared__ __align__(8) unsigned long long bars[kGbWarps * kGbDepth];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    pdl_trigger();
    const uint32_t ring = (uint32_t)__cvta_generic_to_shared(gb_smem) + (uint32_t)warp * (kGbDepth * kGbSlot);
    const uint32_t bar0 = (uint32_t)__cvta_generic_to_shared(bars) + 8u * (uint32_t)(warp * kGbDepth);
    if (lane == 0) {
#pragma unroll
        for (int d = 0; d < kGbDepth; ++d)
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar0 + 8u * d) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
    pdl_wait();                                     // Y is still being read by the previous step's gradient
    stamp_begin(stamp);
    const int32_t *I = ind ? ind->idx + idx_off : idx;
    const int gw = blockIdx.x * kGbWarps + warp, W = gridDim.x * kGbWarps;
    // rows of A are read once per epoch: they leave L2 first (the Y and G stages of the pipelined graph are what is read again)
    unsigned long long pol_first;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_first));

    // labels (and the range check): one thread per sampled row
    for (int row = blockIdx.x * blockDim.x + threadIdx.x; row < sb; row += gridDim.x * blockDim.x) {
        const int64_t src = I[row];
        const bool ok = src >= 0 && src < m;
        yI[row] = ok ? y[src] : 0.f;
        if (!ok) flag_index_error(err_flag);
    }

    const uint32_t rowB = (uint32_t)n * 2u;                                 // a multiple of 16
    const int ppr = (int)((rowB + kGbSlot - 1) / kGbSlot);                  // pieces per row
    const int my_rows = gw < sb ? (sb - 1 - gw) / W + 1 : 0;                // rows gw, gw + W, ...
    const int total = my_rows * ppr;
    int64_t src_row = 0, src_prev = 0;                                      // lane k: source row of the k-th row of this / the previous batch of 32
    uint32_t phase_bits = 0;                                                // per-slot parity of the full barriers
    // software pipeline over pieces: loads run kGbAhead pieces ahead of the stores; a slot is loaded again
    // kGbDepth - kGbAhead iterations after its store was committed
    for (int p = 0; p < total + kGbAhead; ++p) {
        if (p < total) {
            const int k = p / ppr, piece = p - k * ppr;
            if (piece == 0 && (k & 31) == 0) {                              // a new batch of 32 rows: one index per lane
                const int kk = k + lane;
                src_prev = src_row;
                src_row = kk < my_rows ? (int64_t)I[gw + kk * W] : 0;
            }
            const int64_t src = __shfl_sync(0xffffffffu, src_row, k & 31);
            const bool ok = src >= 0 && src < m;
            const uint32_t off = (uint32_t)piece * kGbSlot, bytes = min(kGbSlot, rowB - off);
            const int slot = p % kGbDepth;
            const uint32_t dst = ring + (uint32_t)slot * kGbSlot, bar = bar0 + 8u * slot;
            if (ok) {
                if (lane == 0) {
                    // the store that last read this slot has finished reading it
                    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(kGbDepth - kGbAhead - 1) : "memory");
                    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                                 ::"r"(dst), "l"(A + src * lda + off / 2), "r"(bytes), "r"(bar), "l"(pol_first) : "memory");
                }
            } else {
                // an out-of-range index reads as a zero row: written by the lanes, nothing goes through the ring
                unsigned char *yrow = reinterpret_cast<unsigned char *>(Y + (int64_t)(gw + k * W) * ldy) + off;
                for (uint32_t e = lane * 16u; e < bytes; e += 512u) *reinterpret_cast<uint4 *>(yrow + e) = make_uint4(0u, 0u, 0u, 0u);
                if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
            }
        }
        const int q = p - kGbAhead;                                         // the piece to store now
        if (q >= 0) {
            const int k = q / ppr, piece = q - k * ppr;
            const int slot = q % kGbDepth;
            const uint32_t srcs = ring + (uint32_t)slot * kGbSlot, bar = bar0 + 8u * slot;
            const uint32_t off = (uint32_t)piece * kGbSlot, bytes = min(kGbSlot, rowB - off);
            const uint32_t parity = (phase_bits >> slot) & 1u;
            phase_bits ^= 1u << slot;
            const int k_load = min(p, total - 1) / ppr;                     // the loads are at most one batch ahead
            const int64_t src = __shfl_sync(0xffffffffu, (k >> 5) == (k_load >> 5) ? src_row : src_prev, k & 31);
            if (lane == 0) {
                uint32_t done;
                do {
                    asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                                 : "=r"(done) : "r"(bar), "r"(parity) : "memory");
                } while (!done);
                if (src >= 0 && src < m) {
                    unsigned char *yrow = reinterpret_cast<unsigned char *>(Y + (int64_t)(gw + k * W) * ldy) + off;
                    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(yrow), "r"(srcs), "r"(bytes) : "memory");
                }
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            }
            __syncwarp();
        }
    }
    if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");   // the stores have landed before the CTA exits
    stamp_end_warp(stamp);
}

cudaError_t gather_configure()
{
    return cudaFuncSetAttribute(gather_bulk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)((size_t)kGbWarps * kGbDepth * kGbSlot));
}

int launch_gather(cudaStream_t st, const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n,
                  const int32_t *idx, const StepParams *ind, int64_t idx_off, int32_t sb, uint16_t *Y, int32_t ldy,
                  float *yI, int *err_flag, int num_sms)
{
    if (n % 8 == 0 && n * 2 >= 512 && ldy == n && (int64_t)sb * n * 2 >= (1 << 20)) {
        const size_t smem = (size_t)kGbWarps * kGbDepth * kGbSlot;
        const int ppr = (n * 2 + (int)kGbSlot - 1) / (int)kGbSlot;
        const int64_t pieces = (int64_t)sb * ppr;
        const int blocks = (int)std::max<int64_t>(1, std::min<int64_t>(num_sms, (pieces + kGbWarps * 2 - 1) / (kGbWarps * 2)));
        launch_pdl(gather_bulk_kernel, dim3(blocks), dim3(32 * kGbWarps), smem, st, 1, A, lda, y, m, n, idx, ind, idx_off, sb, Y,
                   ldy, yI, err_flag, g_stamp);
        return 1;
    }
    const int64_t total = (int64_t)sb * (ldy >> 3);
    const int threads = 256;
    const unsigned blocks = (unsigned)((total + threads - 1) / threads);
    launch_pdl(gather_rows_kernel, dim3(blocks), dim3(threads), 0, st, 1, A, lda, y, m, n, idx, ind, idx_off, sb, Y, ldy, yI,
               err_flag, g_stamp);
    return 1;
}

// x_bf = bf16_rne(x): the margin kernel's view of the weights.
__global__ void shadow_kernel(const float *x, const StepParams *ind, int32_t n,
                              uint16_t *xbf, int32_t ldxb, int split)
{
    pdl_trigger();
    pdl_wait();
    const float *xs = ind ? ind->x : x;
    int32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    store_shadow(xbf, split ? ldxb : 0, k, xs[k]);
    if (!split) xbf[ldxb + k] = xbf[2 * ldxb + k] = 0;      // the residue rows read as zero when the split is off
}

int launch_shadow(cudaStream_t st, const float *x, const StepParams *ind, int32_t n, uint16_t *xbf, int32_t ldxb, int split)
{
    launch_pdl(shadow_kernel, dim3((n + 255) / 256), dim3(256), 0, st, 1, x, ind, n, xbf, ldxb, split);
    return 1;
}

// CASGD_OPT_SNAPSHOT: the iterate as it enters the last step of a graph (tests compare that step with the oracle)
__global__ void snapshot_kernel(const float *x, const StepParams *ind, int32_t n, float *dst)
{
    pdl_trigger();
    pdl_wait();
    const float *xs = ind ? ind->x : x;
    const int32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) dst[k] = ld_dep(xs + k);
}

int launch_snapshot(cudaStream_t st, const float *x, const StepParams *ind, int32_t n, float *dst)
{
    launch_pdl(snapshot_kernel, dim3((n + 255) / 256), dim3(256), 0, st, 1, x, ind, n, dst);
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

int launch_widen(cudaStream_t st, const uint16_t *A, int64_t lda, int64_t m, int32_t n, float *A32, int64_t lda32, int num_sms)
{
    widen_kernel<<<num_sms * 8, 256, 0, st>>>(A, lda, m, n, A32, lda32);
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

int launch_repack(cudaStream_t st, const uint16_t *X, int64_t ldx, int64_t m, int32_t n, uint16_t *A, int64_t lda, int num_sms)
{
    repack_kernel<<<num_sms * 8, 256, 0, st>>>(X, ldx, m, n, A, lda);
    return 1;
}

// CASGD_OPT_STAMPS: fold the {first start, last end} slots of the steps just run into per-stage totals and re-arm them.
__global__ void stamp_collect_kernel(unsigned long long *slots, int nslots, unsigned long long *accum_ns,
                                     unsigned long long *count, unsigned long long *raw_copy)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nslots) return;
    const unsigned long long t0 = slots[2 * i], t1 = slots[2 * i + 1];
    raw_copy[2 * i] = t0;                               // the timeline of the graph just replayed (CASGD_DBG_STAMPS)
    raw_copy[2 * i + 1] = t1;
    if (t1 != 0ull && t0 != ~0ull && t1 >= t0) {
        atomicAdd(accum_ns + (i & 7), t1 - t0);
        atomicAdd(count + (i & 7), 1ull);
    }
    slots[2 * i] = ~0ull;
    slots[2 * i + 1] = 0ull;
}

int launch_stamp_collect(cudaStream_t st, unsigned long long *slots, int nslots, unsigned long long *accum_ns,
                         unsigned long long *count, unsigned long long *raw_copy)
{
    stamp_collect_kernel<<<(nslots + 255) / 256, 256, 0, st>>>(slots, nslots, accum_ns, count, raw_copy);
    return 1;
}

// casgd_outer_steps_host with pinned host buffers and a small step: ONE kernel reads the indices and x straight from the
// mapped host memory (no copy-engine round trips: each cudaMemcpyAsync of 16 KB costs ~5 us of latency on a stream the
// host is waiting for), writes the device stages and builds the BF16 shadow; a second one writes x back after the steps.
__global__ void __launch_bounds__(256)
stage_in_kernel(const int32_t *idx_host, int64_t count, int32_t *idx_stage, const float *x_host, int32_t n, float *x_stage,
                uint16_t *xbf, int32_t ldxb, int split)
{
    pdl_trigger();
    pdl_wait();
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, T = (int64_t)gridDim.x * blockDim.x;
    for (int64_t k = t; k < count; k += T) idx_stage[k] = idx_host[k];
    for (int64_t k = t; k < n; k += T) {
        const float v = x_host[k];
        x_stage[k] = v;
        store_shadow(xbf, split ? ldxb : 0, (int32_t)k, v);
        if (!split) xbf[ldxb + k] = xbf[2 * ldxb + k] = 0;
    }
}

__global__ void __launch_bounds__(256)
stage_out_kernel(const float *x_stage, int32_t n, float *x_host)
{
    pdl_trigger();
    pdl_wait();
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) x_host[k] = ld_dep(x_stage + k);
}

int launch_stage_in(cudaStream_t st, const int32_t *idx_host, int64_t count, int32_t *idx_stage, const float *x_host, int32_t n,
                    float *x_stage, uint16_t *xbf, int32_t ldxb, int split)
{
    const int64_t work = std::max<int64_t>(count, n);
    const int blocks = (int)std::min<int64_t>(148, (work + 255) / 256);
    launch_pdl(stage_in_kernel, dim3(blocks), dim3(256), 0, st, 1, idx_host, count, idx_stage, x_host, n, x_stage, xbf, ldxb, split);
    return 1;
}

int launch_stage_out(cudaStream_t st, const float *x_stage, int32_t n, float *x_host)
{
    launch_pdl(stage_out_kernel, dim3(std::min(148, (n + 255) / 256)), dim3(256), 0, st, 1, x_stage, n, x_host);
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

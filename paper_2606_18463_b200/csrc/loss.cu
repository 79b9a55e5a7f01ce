// loss.cu -- F(x) = (1/m) sum_i L(a_i^T x, y_i): one streaming pass over the BF16 matrix A.
// A pure HBM-bound GEMV (2 m n bytes, the "GEMV HBM GB/s" of BASELINE.json:metric).
//
// loss_stream_kernel: one persistent CTA per SM, 16 warps, and every warp runs its OWN pipeline: lane 0 issues
// 1-D bulk copies (cp.async.bulk, the TMA engine) of contiguous pieces of A into a private ring of kLsDepth
// 4 KB shared-memory slots, each with its own mbarrier, and the 32 lanes consume a slot while the next two are
// in flight (128 KB of reads outstanding per SM; no cross-warp synchronisation at all). x sits in shared memory
// as FP32; margins and per-row losses are FP32, the sum is FP64; two rows are processed together so that every
// x value read from shared memory is used several times. Deterministic reduction: per-CTA partials, added in a
// fixed order by the last CTA to finish.
//   MODE 0  rows of at most 1 KB whose stride is a multiple of 16 B: a slot holds 4 k whole rows plus their labels
//           (two copies); GS lanes share a group of 4 rows, 32/GS groups at a time.
//   MODE 1  wider rows: a slot holds a 2 KB segment of each of two consecutive rows (two copies); the lane
//           accumulators carry over the segments of a row pair.
//   MODE 2  narrow rows with an unaligned stride (n = 18: 36-byte rows, read from the caller's own X, not from
//           the padded copy: 36 instead of 64 bytes per row): a slot holds 32 k whole rows plus their labels, one
//           lane per row.
// loss_rows_kernel (plain 16-byte loads, x from global memory) remains for n > kLsMaxN.
#include <algorithm>

#include "common.cuh"

namespace casgd {

namespace {

constexpr int kLsWarps = 16;
constexpr int kLsThreads = 32 * kLsWarps;
constexpr int kLsDepth = 3;
constexpr uint32_t kLsSlot = 4096;
constexpr uint32_t kLsSeg = kLsSlot / 2;
constexpr uint32_t kLsYBytes = 512;                  // labels of the rows of a slot (MODE 0 / 2: at most 128 rows)
constexpr uint32_t kLsSlotY = kLsSlot + kLsYBytes;
constexpr int kLsMaxN = 8192;                        // x in shared memory as FP32: 32 KB

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    do {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ uint4 lds_u4(uint32_t saddr)
{
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(saddr));
    return v;
}
__device__ __forceinline__ float4 lds_f4(uint32_t saddr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(saddr));
    return v;
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t saddr)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(saddr));
    return v;
}
__device__ __forceinline__ uint32_t lds_u16(uint32_t saddr)
{
    uint32_t v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=r"(v) : "r"(saddr));
    return v;
}
__device__ __forceinline__ float lds_f32(uint32_t saddr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(saddr));
    return v;
}

// keep the first `valid` (< 8) BF16 of a 16-byte vector, zero the rest (pad columns may hold anything)
__device__ __forceinline__ uint4 mask_tail(uint4 v, int valid)
{
    uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        if (2 * q >= valid) w[q] = 0u;
        else if (2 * q + 1 >= valid) w[q] &= 0x0000ffffu;
    }
    return make_uint4(w[0], w[1], w[2], w[3]);
}

// Fill one slot from global memory: a bulk copy when the piece is a multiple of 16 bytes (always, except
// possibly the very last piece of the matrix), else by the lanes themselves. Completes `bar` either way.
__device__ __forceinline__ void fill_piece(uint32_t dst, const uint16_t *src, uint32_t bytes, uint32_t bar, int lane,
                                           bool first_of_slot, bool last_of_slot, uint32_t slot_bytes_total)
{
    if ((slot_bytes_total & 15u) == 0u) {
        if (lane == 0) {
            if (first_of_slot) mbar_expect_tx(bar, slot_bytes_total);
            bulk_g2s(dst, src, bytes, bar);
        }
    } else {
        for (uint32_t e = lane; e < bytes / 2; e += 32) {
            const uint32_t v = src[e];
            asm volatile("st.shared.u16 [%0], %1;" ::"r"(dst + 2u * e), "h"((uint16_t)v) : "memory");
        }
        __syncwarp();
        if (lane == 0 && last_of_slot) mbar_arrive(bar);
    }
}

template <int MODE>
__global__ void __launch_bounds__(kLsThreads, 1)
loss_stream_kernel(const uint16_t *__restrict__ A, int64_t ld, const float *__restrict__ y, int64_t m, int32_t n, int loss,
                   const float *__restrict__ x, int32_t rows_per_slot, int32_t gs, double *__restrict__ block_partials,
                   unsigned *__restrict__ done, double *__restrict__ result)
{
    extern __shared__ __align__(128) unsigned char ls_smem[];
    __shared__ double warp_part[kLsWarps];
    __shared__ __align__(8) unsigned long long bars[kLsWarps * kLsDepth];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nvec = (n + 7) >> 3;
    const int xpad = nvec * 8;
    float *xs = reinterpret_cast<float *>(ls_smem);
    for (int k = threadIdx.x; k < xpad; k += kLsThreads) xs[k] = (k < n) ? x[k] : 0.f;
    const uint32_t xs_a = smem_u32(xs);
    const uint32_t ring = ((xs_a + 4u * (uint32_t)xpad + 127u) & ~127u) + (uint32_t)warp * (kLsDepth * (MODE == 1 ? kLsSlot : kLsSlotY));
    const uint32_t bar0 = smem_u32(bars) + 8u * (uint32_t)(warp * kLsDepth);
    if (lane == 0) {
#pragma unroll
        for (int d = 0; d < kLsDepth; ++d) mbar_init(bar0 + 8u * d, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    float xr[MODE == 2 ? 32 : 1];
    const bool x_in_regs = MODE == 2 && n <= 32 && (n & 1) == 0 && (ld & 1) == 0;
    if (MODE == 2) {
#pragma unroll
        for (int k = 0; k < 32; ++k) xr[k] = (x_in_regs && k < n) ? xs[k] : 0.f;
    }
    const int64_t gw = (int64_t)blockIdx.x * kLsWarps + warp;          // global warp id
    const int64_t W = (int64_t)gridDim.x * kLsWarps;
    const uint32_t rowB = (uint32_t)(ld * 2);
    double local = 0.0;

    if (MODE == 0 || MODE == 2) {
        // unit = rows_per_slot consecutive whole rows (one contiguous piece) + their labels (a second piece)
        const int64_t nunits = (m + rows_per_slot - 1) / rows_per_slot;
        // running state of the producer and of the consumer: this warp's next unit and where it starts (the 64-bit
        // products per slot were a quarter of the narrow-row kernel's instructions)
        const int64_t unit_stride_rows = W * rows_per_slot;
        const uint32_t full_bytes = (uint32_t)rows_per_slot * rowB, full_ybytes = 4u * (uint32_t)rows_per_slot;
        const bool full_ok = ((full_bytes | full_ybytes) & 15u) == 0u;
        int64_t p_unit = gw;
        const uint16_t *p_src = A + gw * rows_per_slot * ld;
        const float *p_y = y + gw * rows_per_slot;
        auto issue = [&](int slot) {
            if (p_unit >= nunits) return;
            const uint32_t dst = ring + (uint32_t)slot * kLsSlotY, bar = bar0 + 8u * slot;
            if (p_unit + 1 < nunits && full_ok) {       // a whole unit: two bulk copies
                if (lane == 0) {
                    mbar_expect_tx(bar, full_bytes + full_ybytes);
                    bulk_g2s(dst, p_src, full_bytes, bar);
                    bulk_g2s(dst + kLsSlot, p_y, full_ybytes, bar);
                }
            } else {
                const int64_t row0 = p_unit * rows_per_slot;
                const int rows = (int)min((int64_t)rows_per_slot, m - row0);
                // the last row of the matrix ends at its n-th element (rounded up to the 16-byte vector when aligned)
                uint32_t bytes = (uint32_t)rows * rowB;
                if (row0 + rows == m) bytes = (uint32_t)(rows - 1) * rowB + (MODE == 0 ? (uint32_t)xpad * 2u : (uint32_t)n * 2u);
                const uint32_t ybytes = 4u * (uint32_t)rows;
                const uint32_t total = (((bytes | ybytes) & 15u) == 0u) ? bytes + ybytes : 1u;   // odd total: copied by the lanes
                fill_piece(dst, p_src, bytes, bar, lane, true, false, total);
                fill_piece(dst + kLsSlot, reinterpret_cast<const uint16_t *>(p_y), ybytes, bar, lane, false, true, total);
            }
            p_unit += W;
            p_src += unit_stride_rows * ld;
            p_y += unit_stride_rows;
        };
#pragma unroll 1
        for (int d = 0; d < kLsDepth - 1; ++d) issue(d);
        int slot = 0;
        uint32_t phase = 0;
#pragma unroll 1
        for (int64_t unit = gw; unit < nunits; unit += W) {
            issue(slot == 0 ? kLsDepth - 1 : slot - 1);                         // into the slot consumed last iteration
            const int rows = unit + 1 < nunits ? rows_per_slot : (int)(m - unit * rows_per_slot);
            const uint32_t sbase = ring + (uint32_t)slot * kLsSlotY;
            mbar_wait(bar0 + 8u * slot, phase);
            if (MODE == 0) {
                // gs (>= 4) lanes share a group of 4 rows: every x vector read from shared memory serves 4 rows;
                // a transposed shuffle reduction leaves the total of row q of the group in quarter q of its lanes
                const int g = lane / gs, l = lane % gs, ng = 32 / gs, qw = gs >> 2;
                const int trips = (rows + 4 * ng - 1) / (4 * ng);       // same trip count for every lane
#pragma unroll 1
                for (int t = 0; t < trips; ++t) {
                    const int rbase = 4 * (g + t * ng);
                    uint32_t ra[4];
#pragma unroll
                    for (int i = 0; i < 4; ++i) ra[i] = sbase + (uint32_t)min(rbase + i, rows - 1) * rowB;
                    float acc[4] = {0.f, 0.f, 0.f, 0.f};
                    for (int cv = l; cv < nvec; cv += gs) {
                        const float4 x0 = lds_f4(xs_a + 32u * cv), x1 = lds_f4(xs_a + 32u * cv + 16u);
                        const bool tail = cv * 8 + 8 > n;
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            uint4 a = lds_u4(ra[i] + 16u * cv);
                            if (tail) a = mask_tail(a, n - cv * 8);
                            acc[i] = dot8(a, x0, x1, acc[i]);
                        }
                    }
                    const bool hi = l & (gs >> 1), hq = l & qw;
                    float k0 = hi ? acc[2] : acc[0], k1 = hi ? acc[3] : acc[1];
                    k0 += __shfl_xor_sync(0xffffffffu, hi ? acc[0] : acc[2], gs >> 1);
                    k1 += __shfl_xor_sync(0xffffffffu, hi ? acc[1] : acc[3], gs >> 1);
                    float k = hq ? k1 : k0;
                    k += __shfl_xor_sync(0xffffffffu, hq ? k0 : k1, qw);
                    for (int o = qw >> 1; o > 0; o >>= 1) k += __shfl_xor_sync(0xffffffffu, k, o);
                    const int row = rbase + l / qw;                     // quarter q of the lanes holds row q
                    if ((l & (qw - 1)) == 0 && row < rows)
                        local += (double)loss_value_rt(loss, k, lds_f32(sbase + kLsSlot + 4u * (uint32_t)row));
                }
            } else {
                // one lane per row; rows are 2-byte aligned (4-byte when ld is even)
                const int trips = (rows + 31) >> 5;
#pragma unroll 1
                for (int t = 0; t < trips; ++t) {
                    const int rr = lane + 32 * t;
                    if (rr < rows) {
                        const uint32_t ra = sbase + (uint32_t)rr * rowB;
                        float acc = 0.f, acc2 = 0.f;
                        if (x_in_regs) {
                            // n <= 32 and even: x lives in registers; the row's n / 2 words in blocks of four under
                            // UNIFORM branches (a predicated-off load or FMA still takes its issue slot, and this
                            // kernel is issue-bound at n = 18: 16 predicated words were 106 of its 173 instructions
                            // per 32 rows)
                            const int nw = n >> 1;
#pragma unroll
                            for (int kb = 0; kb < 16; kb += 4) {
                                if (kb < nw) {
                                    if (kb + 4 <= nw) {
                                        uint32_t w[4];
#pragma unroll
                                        for (int k = 0; k < 4; ++k) w[k] = lds_u32(ra + 4u * (kb + k));
#pragma unroll
                                        for (int k = 0; k < 4; ++k) {
                                            acc = fmaf(bf16lo(w[k]), xr[2 * (kb + k)], acc);
                                            acc2 = fmaf(bf16hi(w[k]), xr[2 * (kb + k) + 1], acc2);
                                        }
                                    } else {
#pragma unroll
                                        for (int k = 0; k < 3; ++k) {
                                            if (kb + k < nw) {
                                                const uint32_t w = lds_u32(ra + 4u * (kb + k));
                                                acc = fmaf(bf16lo(w), xr[2 * (kb + k)], acc);
                                                acc2 = fmaf(bf16hi(w), xr[2 * (kb + k) + 1], acc2);
                                            }
                                        }
                                    }
                                }
                            }
                        } else if ((ld & 1) == 0) {
                            const int nw = n >> 1;
#pragma unroll 3
                            for (int k = 0; k < nw; ++k) {
                                const uint32_t w = lds_u32(ra + 4u * k);
                                acc = fmaf(bf16lo(w), lds_f32(xs_a + 8u * k), acc);
                                acc2 = fmaf(bf16hi(w), lds_f32(xs_a + 8u * k + 4u), acc2);
                            }
                            if (n & 1) acc = fmaf(__uint_as_float(lds_u16(ra + 2u * (n - 1)) << 16), lds_f32(xs_a + 4u * (n - 1)), acc);
                        } else {
                            for (int k = 0; k < n; ++k)
                                acc = fmaf(__uint_as_float(lds_u16(ra + 2u * k) << 16), lds_f32(xs_a + 4u * k), acc);
                        }
                        local += (double)loss_value_rt(loss, acc + acc2, lds_f32(sbase + kLsSlot + 4u * (uint32_t)rr));
                    }
                }
            }
            __syncwarp();                               // every lane is done with the slot before it is refilled
            if (++slot == kLsDepth) { slot = 0; phase ^= 1u; }
        }
    } else {
        // MODE 1: unit = (row pair, 2 KB segment of both rows)
        const uint32_t validB = (uint32_t)xpad * 2u;                    // bytes of a row that hold data (16-byte granules)
        const int nseg = (int)((validB + kLsSeg - 1) / kLsSeg);
        const int64_t npairs = (m + 1) >> 1;
        const int64_t my_pairs = gw < npairs ? (npairs - 1 - gw) / W + 1 : 0;
        const int64_t nunits = my_pairs * nseg;
        auto issue = [&](int64_t u, int slot) {
            if (u >= nunits) return;
            const int64_t pr = gw + (u / nseg) * W;
            const int sg = (int)(u % nseg);
            const uint32_t off = (uint32_t)sg * kLsSeg;
            const uint32_t bytes = min(kLsSeg, validB - off);
            const bool two = 2 * pr + 1 < m;
            const uint32_t dst = ring + (uint32_t)slot * kLsSlot;
            const uint16_t *src = A + 2 * pr * ld + off / 2;
            fill_piece(dst, src, bytes, bar0 + 8u * slot, lane, true, !two, two ? 2u * bytes : bytes);
            if (two) fill_piece(dst + kLsSeg, src + ld, bytes, bar0 + 8u * slot, lane, false, true, 2u * bytes);
        };
#pragma unroll 1
        for (int d = 0; d < kLsDepth - 1; ++d) issue(d, d);
        int slot = 0;
        uint32_t phase = 0;
        float acc0 = 0.f, acc1 = 0.f, y0 = 0.f, y1 = 0.f, yn0 = 0.f, yn1 = 0.f;
        if (lane == 0 && gw < npairs) {
            yn0 = __ldg(y + 2 * gw);
            yn1 = (2 * gw + 1 < m) ? __ldg(y + 2 * gw + 1) : 0.f;
        }
#pragma unroll 1
        for (int64_t u = 0; u < nunits; ++u) {
            issue(u + kLsDepth - 1, slot == 0 ? kLsDepth - 1 : slot - 1);
            const int64_t pr = gw + (u / nseg) * W;
            const int sg = (int)(u % nseg);
            if (sg == 0 && lane == 0) {                 // labels travel one row pair ahead of their use
                y0 = yn0;
                y1 = yn1;
                const int64_t nx = pr + W;
                if (nx < npairs) {
                    yn0 = __ldg(y + 2 * nx);
                    yn1 = (2 * nx + 1 < m) ? __ldg(y + 2 * nx + 1) : 0.f;
                }
            }
            const uint32_t off = (uint32_t)sg * kLsSeg;
            const int vecs = (int)(min(kLsSeg, validB - off) >> 4);
            const int cv0 = (int)(off >> 4);
            const uint32_t sbase = ring + (uint32_t)slot * kLsSlot;
            mbar_wait(bar0 + 8u * slot, phase);
#pragma unroll 2
            for (int v = lane; v < vecs; v += 32) {
                const int cv = cv0 + v;
                uint4 a0 = lds_u4(sbase + 16u * v);
                uint4 a1 = lds_u4(sbase + kLsSeg + 16u * v);
                if (cv * 8 + 8 > n) { a0 = mask_tail(a0, n - cv * 8); a1 = mask_tail(a1, n - cv * 8); }
                const float4 x0 = lds_f4(xs_a + 32u * cv), x1 = lds_f4(xs_a + 32u * cv + 16u);
                acc0 = dot8(a0, x0, x1, acc0);
                acc1 = dot8(a1, x0, x1, acc1);
            }
            if (sg == nseg - 1) {
                acc0 = warp_sum(acc0);
                acc1 = warp_sum(acc1);
                if (lane == 0) {
                    local += (double)loss_value_rt(loss, acc0, y0);
                    if (2 * pr + 1 < m) local += (double)loss_value_rt(loss, acc1, y1);
                }
                acc0 = acc1 = 0.f;
            }
            __syncwarp();
            if (++slot == kLsDepth) { slot = 0; phase ^= 1u; }
        }
    }

    local = warp_sum(local);
    if (lane == 0) warp_part[warp] = local;
    __syncthreads();
    __shared__ bool s_last;
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int w = 0; w < kLsWarps; ++w) tot += warp_part[w];
        block_partials[blockIdx.x] = tot;
        __threadfence();
        s_last = atomicAdd(done, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!s_last) return;
    // the last CTA to finish adds the per-CTA partials in a fixed order (deterministic) and divides by m
    __threadfence();
    double v = 0.0;
    for (int i = threadIdx.x; i < (int)gridDim.x; i += kLsThreads) v += __ldcg(block_partials + i);
    v = warp_sum(v);
    if (lane == 0) warp_part[warp] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int w = 0; w < kLsWarps; ++w) tot += warp_part[w];
        *result = tot / (double)m;
        *done = 0u;
    }
}

}  // namespace

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
                if (c * 8 + 8 > n) {                       // the pad columns of A and the tail of a global x: mask
                    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
                    for (int q = 0; q < 8 && c * 8 + q < n; ++q)
                        acc0 = fmaf((q & 1) ? bf16hi(w[q >> 1]) : bf16lo(w[q >> 1]), xv[c * 8 + q], acc0);
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

static int launch_loss_rows(cudaStream_t st, const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n, int loss,
                            const float *x, double *block_partials, int32_t max_blocks, int num_sms)
{
    const int nvec = (n + 7) >> 3;
    const size_t smem_x = sizeof(float) * (size_t)nvec * 8;
    const int x_in_smem = smem_x <= 96 * 1024;
    const size_t smem = x_in_smem ? smem_x : 0;
    // resident CTAs per SM: 2048 threads / 512, or fewer when x fills shared memory
    int per_sm = 4;
    if (smem > 0) per_sm = (int)std::min<size_t>(4, (200 * 1024) / (smem + 1024));
    per_sm = std::max(per_sm, 1);
    int blocks = std::min(max_blocks, num_sms * per_sm);
    auto go = [&](auto kern, int gs) {
        int64_t rows_per_pass = (int64_t)blocks * kLossThreads / gs;
        if (rows_per_pass > m) blocks = (int)std::max<int64_t>(1, (m * gs + kLossThreads - 1) / kLossThreads);
        kern<<<blocks, kLossThreads, smem, st>>>(A, lda, y, m, n, loss, x, x_in_smem, block_partials);
    };
    if (nvec >= 32) go(loss_rows_kernel<32>, 32);
    else if (nvec > 8) go(loss_rows_kernel<16>, 16);
    else if (nvec > 4) go(loss_rows_kernel<8>, 8);
    else if (nvec > 2) go(loss_rows_kernel<4>, 4);
    else if (nvec > 1) go(loss_rows_kernel<2>, 2);
    else go(loss_rows_kernel<1>, 1);
    return blocks;
}

cudaError_t loss_configure()
{
    // MODE 1 (4 KB slots) takes x up to kLsMaxN floats; MODE 0 / 2 (slots with labels) have n <= 512
    const int cap = (int)(128 + sizeof(float) * kLsMaxN + 128 + (size_t)kLsWarps * kLsDepth * kLsSlot);
    cudaError_t e = cudaFuncSetAttribute(loss_stream_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(loss_stream_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(loss_stream_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap);
    // the plain-load kernel keeps x in shared memory up to 96 KB
    const int xcap = 96 * 1024;
    if (e == cudaSuccess) e = cudaFuncSetAttribute(loss_rows_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, xcap);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(loss_rows_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, xcap);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(loss_rows_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, xcap);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(loss_rows_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, xcap);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(loss_rows_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, xcap);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(loss_rows_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, xcap);
    return e;
}

// A/lda: the library's 16-byte-aligned layout. X/ldx: the caller's own matrix when it was repacked (else null):
// narrow unaligned rows are streamed from there (fewer bytes). impl: 0 = choose, 1 = plain-load kernel.
int launch_loss(cudaStream_t st, const uint16_t *A, int64_t lda, const uint16_t *X, int64_t ldx, const float *y, int64_t m,
                int32_t n, int loss, const float *x, double *block_partials, int32_t max_blocks, double *result_dev,
                unsigned *done_counter, int impl, int num_sms)
{
    int blocks;
    const int nvec = (n + 7) >> 3;
    if (impl == 1 || n > kLsMaxN || max_blocks < num_sms || (uintptr_t)y % 16 != 0) {
        blocks = launch_loss_rows(st, A, lda, y, m, n, loss, x, block_partials, max_blocks, num_sms);
        loss_finish_kernel<<<1, 256, 0, st>>>(block_partials, blocks, m, result_dev);
        return 2;
    } else {
        const size_t fixed = 128 + sizeof(float) * (size_t)nvec * 8 + 128;
        auto go = [&](auto kern, const uint16_t *base, int64_t ld, int rows_per_slot, int gs, int64_t nunits, uint32_t slot_bytes) {
            blocks = (int)std::max<int64_t>(1, std::min<int64_t>(num_sms, (nunits + kLsWarps - 1) / kLsWarps));
            kern<<<blocks, kLsThreads, fixed + (size_t)kLsWarps * kLsDepth * slot_bytes, st>>>(
                base, ld, y, m, n, loss, x, rows_per_slot, gs, block_partials, done_counter, result_dev);
        };
        const bool narrow_ok = X && ((uintptr_t)X % 16 == 0) && (uint64_t)ldx * 2 * 32 <= kLsSlot && ldx * 2 < lda * 2;
        if (narrow_ok) {
            int rps = (int)(kLsSlot / (ldx * 2)) / 32 * 32;             // 32 k rows: pieces of A and of y stay 16-byte aligned
            rps = std::min(rps, (int)kLsYBytes / 4);
            go(loss_stream_kernel<2>, X, ldx, rps, 1, (m + rps - 1) / rps, kLsSlotY);
        } else if ((uint64_t)lda * 2 * 4 <= kLsSlot) {
            int gs = 4;
            while (gs < 32 && gs < nvec) gs <<= 1;
            int rps = (int)(kLsSlot / (lda * 2)) & ~3;                  // a multiple of 4 rows: the labels are a 16-byte-aligned piece
            rps = std::min(rps, (int)kLsYBytes / 4);
            go(loss_stream_kernel<0>, A, lda, rps, gs, (m + rps - 1) / rps, kLsSlotY);
        } else {
            go(loss_stream_kernel<1>, A, lda, 2, 32, (m + 1) / 2, kLsSlot);
        }
    }
    return 1;
}

}  // namespace casgd

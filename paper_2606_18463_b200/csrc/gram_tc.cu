// gram_tc.cu -- Alg. 1 lines 3-4 on the 5th-generation tensor cores:
//   G = Y Y^T (lower-triangular 128x128 tiles only; BF16 operands, FP32 accumulation in TMEM) with the
//   margin r = Y x_bf fused in: on the diagonal tile of each row block the B operand carries 16 extra
//   rows, the first of which is x_bf (BASELINE.json:north_star "carrying x as an extra B-operand column").
//
// One persistent CTA per SM, warp-specialised:
//   warp 0      TMA producer: 128B-swizzled K-major boxes of Y (and of x_bf) into a 5-stage smem ring
//   warp 1      allocates TMEM, then one lane issues tcgen05.mma (M=128, N=128/144/16, K=16, kind::f16)
//   warps 2..5  epilogue: tcgen05.ld the FP32 accumulator (two TMEM slots, so the epilogue of tile i
//               overlaps the MMAs of tile i+1) and store G / r
// G = Y Y^T is a "TN" product: both operands are K-major tiles of the same matrix, so on diagonal tiles
// one smem tile serves as A and as B. Few-tile shapes are split along K (partial sums added with red.f32).
#include <cuda.h>

#include <cstdio>
#include <cstring>

#include "common.cuh"

namespace casgd {

namespace {

constexpr int BM = 128, BN = 128, BK = 64, XR = 16;
constexpr int kStages = 5;
constexpr uint32_t kTileBytes = BM * BK * 2;            // 16384
constexpr uint32_t kXBytes = XR * BK * 2;               // 2048
constexpr uint32_t kStageBytes = 2 * kTileBytes + kXBytes;
constexpr uint32_t kOffB = 0, kOffX = kTileBytes, kOffA = kTileBytes + kXBytes;
constexpr uint32_t kAccCols = 256;                      // TMEM columns per accumulator slot (144 used)
constexpr uint32_t kTmemCols = 512;
constexpr int kThreads = 192;
constexpr int kEpiStride = 36;                          // floats per row of an epilogue transpose buffer (conflict-free)
constexpr uint32_t kEpiBufB = 32 * kEpiStride * 4;       // per epilogue warp
constexpr size_t kSmemBytes = 1024 + (size_t)kStages * kStageBytes + 256 + 4 * kEpiBufB;

struct GramParams {
    float *G;
    float *r;
    int32_t ldg, sb, b, n, T, ntiles, ksplit, kb_total, full_lower;
    int32_t row_base;                   // first row of this step's Y buffer inside the (double-buffered) stage
    int32_t no_margin;                  // pipelined schedule: r is a kernel of its own, no x_bf rows in the B operand
    unsigned long long *stamp;
};

// ------------------------------------------------------------------------------------ PTX ---

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
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *map, uint32_t bar, int32_t c0, int32_t c1)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
                 ::"r"(dst), "l"((uint64_t)map), "r"(bar), "r"(c0), "r"(c1) : "memory");
}
__device__ __forceinline__ bool elect_one()
{
    uint32_t pred;
    asm volatile("{\n.reg .pred P;\nelect.sync _|P, 0xffffffff;\nselp.u32 %0, 1, 0, P;\n}" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_mma_bf16(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc)
{
    asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}"
                 ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void tc_ld32(uint32_t taddr, uint32_t (&v)[32])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                 "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                 "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                   "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
                   "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
                   "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
                 : "r"(taddr) : "memory");
}
__device__ __forceinline__ uint32_t tc_ld1(uint32_t taddr)
{
    uint32_t v;
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(v) : "r"(taddr) : "memory");
    return v;
}
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ float tc_ld_margin(uint32_t taddr)
{
    // the margin's accumulator columns 0..3 = Y . (rows 0..3 of the x_bf operand): row 0 is bf16(x); rows 1 and 2 are
    // zero, or its BF16 residues with CASGD_OPT_MARGIN_SPLIT; row 3 is zero. Their sum is r either way (c + 0 == c).
    uint32_t a, b, c, d;
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(a), "=r"(b), "=r"(c), "=r"(d) : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
    return (__uint_as_float(a) + __uint_as_float(b)) + (__uint_as_float(c) + __uint_as_float(d));
}

// K-major, 128-byte swizzle: rows of 64 BF16 (128 B), 8-row groups 1024 B apart (SBO), descriptor version 1.
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t saddr)
{
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | (1ull << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// kind::f16 instruction descriptor: D = F32, A = B = BF16, both K-major, M = 128, N = n_cols.
__device__ __forceinline__ uint32_t umma_idesc(uint32_t n_cols)
{
    return (1u << 4) | (1u << 7) | (1u << 10) | ((n_cols >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
}

// ------------------------------------------------------------------------- work decoding ---

struct Work {
    int ti, tj, kb0, kb1;
    bool diag, need_g, skip;
};

__device__ __forceinline__ Work decode_work(const GramParams &p, int w)
{
    Work k;
    const int t = w % p.ntiles, ks = w / p.ntiles;
    if (t < p.T) {
        k.ti = k.tj = t;
        k.diag = true;
    } else {
        const int q = t - p.T;                          // strictly-lower tiles: q = ti (ti - 1) / 2 + tj, ti >= 1
        int ti = (int)((1.f + sqrtf(1.f + 8.f * (float)q)) * 0.5f);
        while (ti * (ti - 1) / 2 > q) --ti;
        while ((ti + 1) * ti / 2 <= q) ++ti;
        k.ti = ti;
        k.tj = q - ti * (ti - 1) / 2;
        k.diag = false;
    }
    const int last_row = min(k.ti * BM + BM, p.sb) - 1;
    k.need_g = p.full_lower || (last_row / p.b) > ((k.tj * BN) / p.b);      // holds an entry of a block below the block diagonal
    k.skip = !k.need_g && (!k.diag || p.no_margin);
    k.kb0 = (int)(((int64_t)ks * p.kb_total) / p.ksplit);
    k.kb1 = (int)(((int64_t)(ks + 1) * p.kb_total) / p.ksplit);
    return k;
}

// ------------------------------------------------------------------------------- kernel ---

__global__ void __launch_bounds__(kThreads, 1)
gram_tc_kernel(const __grid_constant__ CUtensorMap tmY, const __grid_constant__ CUtensorMap tmX, const GramParams p)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_base = smem_base + kStages * kStageBytes;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (kStages + s); };
    auto accf_bar = [&](int s) { return bar_base + 8u * (2 * kStages + s); };
    auto acce_bar = [&](int s) { return bar_base + 8u * (2 * kStages + 2 + s); };
    const uint32_t tmem_slot = bar_base + 8u * (2 * kStages + 4);
    volatile uint32_t *tmem_slot_ptr =
        reinterpret_cast<volatile uint32_t *>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nwork = p.ntiles * p.ksplit;
    pdl_trigger();

    if (warp == 0 && lane == 0) {
        for (int s = 0; s < kStages; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(accf_bar(s), 1); mbar_init(acce_bar(s), 4); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"((uint64_t)&tmY) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"((uint64_t)&tmX) : "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(kTmemCols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;
    pdl_wait();                                     // Y and x_bf come from the gather / the previous gradient
    stamp_begin(p.stamp);

    if (warp == 0) {
        // ===== TMA producer =====
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int w = blockIdx.x; w < nwork; w += gridDim.x) {
                const Work k = decode_work(p, w);
                if (k.skip) continue;
                for (int kb = k.kb0; kb < k.kb1; ++kb) {
                    mbar_wait(empty_bar(stage), phase ^ 1u);
                    const uint32_t sbase = smem_base + stage * kStageBytes;
                    if (k.diag) {
                        mbar_expect_tx(full_bar(stage), kTileBytes + (p.no_margin ? 0u : kXBytes));
                        tma_load_2d(sbase + kOffB, &tmY, full_bar(stage), kb * BK, p.row_base + k.ti * BM);
                        if (!p.no_margin) tma_load_2d(sbase + kOffX, &tmX, full_bar(stage), kb * BK, 0);
                    } else {
                        mbar_expect_tx(full_bar(stage), 2 * kTileBytes);
                        tma_load_2d(sbase + kOffB, &tmY, full_bar(stage), kb * BK, p.row_base + k.tj * BN);
                        tma_load_2d(sbase + kOffA, &tmY, full_bar(stage), kb * BK, p.row_base + k.ti * BM);
                    }
                    if (++stage == kStages) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer: the whole warp runs the loops (uniform control flow keeps the descriptors in uniform
        // registers), one elected lane issues. With a lane-0-only branch every operand is a per-thread register
        // that has to be moved to a uniform register around each tcgen05.mma (measured: ~2x the 64-cycle floor). =====
        {
            int stage = 0;
            uint32_t phase = 0;
            int it = 0;
            for (int w = blockIdx.x; w < nwork; w += gridDim.x) {
                const Work k = decode_work(p, w);
                if (k.skip) continue;
                const int slot = it & 1;
                const uint32_t acc_phase = (uint32_t)(it >> 1) & 1u;
                ++it;
                mbar_wait(acce_bar(slot), acc_phase ^ 1u);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + slot * kAccCols;
                // diagonal tile: A = B = the same smem tile; N = 144 (G tile + margin rows) or 16 (margin only)
                const uint32_t ncols = k.diag ? (k.need_g ? (uint32_t)(BN + (p.no_margin ? 0 : XR)) : (uint32_t)XR) : (uint32_t)BN;
                const uint32_t idesc = umma_idesc(ncols);
                const uint32_t offa = k.diag ? kOffB : kOffA, offb = (k.diag && !k.need_g) ? kOffX : kOffB;
                for (int kb = k.kb0; kb < k.kb1; ++kb) {
                    mbar_wait(full_bar(stage), phase);
                    tc_fence_after();
                    const uint32_t sbase = smem_base + stage * kStageBytes;
                    const uint64_t adesc = umma_desc_sw128(sbase + offa);
                    const uint64_t bdesc = umma_desc_sw128(sbase + offb);
                    const int kcols = min(p.n - kb * BK, BK);
                    const int ksteps = (kcols + 15) >> 4;                  // zero-filled K tail beyond n is skipped
                    const uint32_t first = kb > k.kb0 ? 1u : 0u;
                    if (elect_one()) {
                        if (ksteps == 4) {                                 // a full K block: straight-line issue
                            tc_mma_bf16(d_tmem, adesc, bdesc, idesc, first);
                            tc_mma_bf16(d_tmem, adesc + 2u, bdesc + 2u, idesc, 1u);
                            tc_mma_bf16(d_tmem, adesc + 4u, bdesc + 4u, idesc, 1u);
                            tc_mma_bf16(d_tmem, adesc + 6u, bdesc + 6u, idesc, 1u);
                        } else {
                            for (int ks = 0; ks < ksteps; ++ks)
                                tc_mma_bf16(d_tmem, adesc + 2u * ks, bdesc + 2u * ks, idesc, ks > 0 ? 1u : first);
                        }
                        tc_commit(empty_bar(stage));                       // frees the smem slot when the MMAs retire
                        if (kb == k.kb1 - 1) tc_commit(accf_bar(slot));    // accumulator ready for the epilogue
                    }
                    __syncwarp();
                    if (++stage == kStages) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else {
        // ===== epilogue warps: TMEM lane group (warp % 4), one accumulator row per thread =====
        const int q = warp & 3;
        int it = 0;
        const bool accumulate = p.ksplit > 1;
        const uint32_t ebuf = bar_base + 256 + (uint32_t)(warp - 2) * kEpiBufB;
        for (int w = blockIdx.x; w < nwork; w += gridDim.x) {
            const Work k = decode_work(p, w);
            if (k.skip) continue;
            const int slot = it & 1;
            const uint32_t acc_phase = (uint32_t)(it >> 1) & 1u;
            ++it;
            mbar_wait(accf_bar(slot), acc_phase);
            tc_fence_after();
            const uint32_t t_row = tmem_base + ((uint32_t)(q * 32) << 16) + slot * kAccCols;
            const int row = k.ti * BM + q * 32 + lane;
            const bool row_ok = row < p.sb;
            if (k.need_g) {
#pragma unroll 1
                for (int c = 0; c < BN / 32; ++c) {
                    uint32_t v[32];
                    tc_ld32(t_row + c * 32, v);
                    tc_wait_ld();
                    // transpose through shared memory so that every store instruction writes whole 128-byte lines
#pragma unroll
                    for (int e = 0; e < 32; e += 4)
                        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(ebuf + (uint32_t)(lane * kEpiStride + e) * 4u),
                                     "r"(v[e]), "r"(v[e + 1]), "r"(v[e + 2]), "r"(v[e + 3]) : "memory");
                    __syncwarp();
                    const int c4 = (lane & 7) * 4;
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const int rl = 4 * i + (lane >> 3);
                        uint32_t o0, o1, o2, o3;
                        asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(o0), "=r"(o1), "=r"(o2), "=r"(o3)
                                     : "r"(ebuf + (uint32_t)(rl * kEpiStride + c4) * 4u) : "memory");
                        const int orow = k.ti * BM + q * 32 + rl;
                        if (orow < p.sb) {
                            float *dst = p.G + (int64_t)orow * p.ldg + k.tj * BN + c * 32 + c4;
                            if (!accumulate) *reinterpret_cast<uint4 *>(dst) = make_uint4(o0, o1, o2, o3);
                            else asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst), "f"(__uint_as_float(o0)),
                                              "f"(__uint_as_float(o1)), "f"(__uint_as_float(o2)), "f"(__uint_as_float(o3)) : "memory");
                        }
                    }
                    __syncwarp();
                }
            }
            if (k.diag && !p.no_margin) {
                const float rv = tc_ld_margin(t_row + (k.need_g ? BN : 0));
                if (row_ok) {
                    if (!accumulate) p.r[row] = rv;
                    else atomicAdd(p.r + row, rv);
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(acce_bar(slot));
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(kTmemCols) : "memory");
    }
    stamp_end(p.stamp);
}

// ------------------------------------------------------------------ narrow rows: gather + Gram in one kernel ---
// For n <= 64 (configs[0], configs[1]) a Gram tile has ONE K block and the step is pure latency, so the gather
// (Alg. 1 line 2) and the Gram + margin (lines 3-4) are one kernel with one CTA per 128x128 tile: its 128 threads
// read the tile's row indices, pull the rows straight from A with 16-byte loads and write them into shared memory
// in the 128-byte-swizzled K-major layout tcgen05 expects (chunk c of row r at r * 128 + ((c ^ (r & 7)) << 4)) --
// no TMA descriptor, no Y round trip through L2 before the MMA. Diagonal tiles also write the Y stage and y_I
// (the gradient's second pass and casgd_debug_export read them) and carry x_bf as 16 extra B rows for the margin.
constexpr int kNwThreads = 128;
constexpr uint32_t kNwOffT0 = 0, kNwOffX = kTileBytes, kNwOffT1 = kTileBytes + kXBytes;
constexpr size_t kNwSmem = 1024 + 2 * kTileBytes + kXBytes + 64 + 4 * kEpiBufB;

struct NarrowParams {
    const uint16_t *A;
    int64_t lda, m;
    const float *y;
    const int32_t *idx;
    const StepParams *ind;
    int64_t idx_off;
    const uint16_t *xbf;
    int32_t ldxb;
    uint16_t *Y;
    float *yI, *G, *r;
    int *err_flag;
    int32_t ldy, ldg, sb, b, n, T, full_lower;
    int32_t s1_loss;                    // >= 0 (s = 1): the epilogue also writes z = r and u = l'(r, y_I)
    float *z, *u;
    unsigned long long *stamp;
};

__global__ void __launch_bounds__(kNwThreads)
gram_narrow_kernel(const NarrowParams p)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar = smem_base + 2 * kTileBytes + kXBytes, tmem_slot = bar + 8u;
    const uint32_t ebuf0 = bar + 64u;
    volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(smem_raw + (tmem_slot - smem_u32(smem_raw)));
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    pdl_trigger();

    // tile of this CTA: the T diagonal tiles first, then the strictly lower ones
    int ti, tj;
    if ((int)blockIdx.x < p.T) {
        ti = tj = blockIdx.x;
    } else {
        const int q = (int)blockIdx.x - p.T;
        ti = (int)((1.f + sqrtf(1.f + 8.f * (float)q)) * 0.5f);
        while (ti * (ti - 1) / 2 > q) --ti;
        while ((ti + 1) * ti / 2 <= q) ++ti;
        tj = q - ti * (ti - 1) / 2;
    }
    const bool diag = ti == tj;
    const int last_row = min(ti * BM + BM, p.sb) - 1;
    const bool need_g = p.full_lower || (last_row / p.b) > ((tj * BN) / p.b);
    if (!diag && !need_g) return;

    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(256u) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    pdl_wait();                                     // x_bf and the Y stage belong to the previous step until now
    stamp_begin(p.stamp);

    // ---- gather: thread t owns row t of each operand tile
    const int32_t *I = p.ind ? p.ind->idx + p.idx_off : p.idx;
    const int ksteps = (p.n + 15) >> 4;             // K = 16 steps that hold data
    const int nfill = 2 * ksteps;                   // 16-byte chunks of a tile row the MMAs read
    float ylab = 0.f;                               // label of row ti * 128 + threadIdx.x (diagonal tiles)
    for (int op = 0; op < (diag ? 1 : 2); ++op) {
        const int trow = (op == 0 ? ti : tj) * BM + (int)threadIdx.x;
        int64_t src = -1;
        if (trow < p.sb) {
            src = I[trow];
            if (src < 0 || src >= p.m) { src = -1; if (diag) flag_index_error(p.err_flag); }
        }
        const uint32_t trow_s = smem_base + (op == 0 ? kNwOffT0 : kNwOffT1) + threadIdx.x * 128u;
        uint4 v[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            v[c] = make_uint4(0u, 0u, 0u, 0u);
            if (c < nfill && src >= 0 && c * 8 < p.n) {
                v[c] = ldg_nc_v4(p.A + src * p.lda + c * 8);
                const int valid = p.n - c * 8;
                if (valid < 8) {
                    uint32_t w[4] = {v[c].x, v[c].y, v[c].z, v[c].w};
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        if (2 * q >= valid) w[q] = 0u;
                        else if (2 * q + 1 >= valid) w[q] &= 0x0000ffffu;
                    }
                    v[c] = make_uint4(w[0], w[1], w[2], w[3]);
                }
            }
        }
#pragma unroll
        for (int c = 0; c < 8; ++c)
            if (c < nfill)
                asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(trow_s + (uint32_t)((c ^ (threadIdx.x & 7)) << 4)),
                             "r"(v[c].x), "r"(v[c].y), "r"(v[c].z), "r"(v[c].w) : "memory");
        if (diag && trow < p.sb) {                  // the Y stage and the labels of these 128 rows
#pragma unroll
            for (int c = 0; c < 8; ++c)
                if (c * 8 < p.ldy) *reinterpret_cast<uint4 *>(p.Y + (int64_t)trow * p.ldy + c * 8) = v[c];
            ylab = src >= 0 ? p.y[src] : 0.f;
            p.yI[trow] = ylab;
        }
    }
    if (diag) {                                     // x_bf: 16 rows x 64 columns right behind the B tile (rows 1..15 are zero)
        const int xr = threadIdx.x >> 3, c = threadIdx.x & 7;
        uint4 v = make_uint4(0u, 0u, 0u, 0u);
        if (c * 8 < p.ldxb) v = *reinterpret_cast<const uint4 *>(p.xbf + (int64_t)xr * p.ldxb + c * 8);
        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(smem_base + kNwOffX + (uint32_t)xr * 128u + (uint32_t)((c ^ (xr & 7)) << 4)),
                     "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> visible to the tensor core
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    // ---- MMA: one K block
    if (warp == 0) {
        const uint32_t ncols = diag ? (need_g ? (uint32_t)(BN + XR) : (uint32_t)XR) : (uint32_t)BN;
        const uint32_t idesc = umma_idesc(ncols);
        const uint64_t adesc = umma_desc_sw128(smem_base + kNwOffT0);
        const uint64_t bdesc = umma_desc_sw128(smem_base + (diag ? (need_g ? kNwOffT0 : kNwOffX) : kNwOffT1));
        if (elect_one()) {
            for (int ks = 0; ks < ksteps; ++ks) tc_mma_bf16(tmem_base, adesc + 2u * ks, bdesc + 2u * ks, idesc, ks > 0 ? 1u : 0u);
            tc_commit(bar);
        }
        __syncwarp();
    }
    mbar_wait(bar, 0u);
    tc_fence_after();

    // ---- epilogue: TMEM lane group = warp; transposed through shared memory, whole-line stores
    const uint32_t t_row = tmem_base + ((uint32_t)(warp * 32) << 16);
    const uint32_t ebuf = ebuf0 + (uint32_t)warp * kEpiBufB;
    if (need_g) {
#pragma unroll 1
        for (int c = 0; c < BN / 32; ++c) {
            if (tj * BN + c * 32 > last_row) break;   // columns beyond the tile's last row are above the diagonal
            uint32_t v[32];
            tc_ld32(t_row + c * 32, v);
            tc_wait_ld();
#pragma unroll
            for (int e = 0; e < 32; e += 4)
                asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(ebuf + (uint32_t)(lane * kEpiStride + e) * 4u),
                             "r"(v[e]), "r"(v[e + 1]), "r"(v[e + 2]), "r"(v[e + 3]) : "memory");
            __syncwarp();
            const int c4 = (lane & 7) * 4;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int rl = 4 * i + (lane >> 3);
                uint32_t o0, o1, o2, o3;
                asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(o0), "=r"(o1), "=r"(o2), "=r"(o3)
                             : "r"(ebuf + (uint32_t)(rl * kEpiStride + c4) * 4u) : "memory");
                const int orow = ti * BM + warp * 32 + rl;
                if (orow < p.sb)
                    *reinterpret_cast<uint4 *>(p.G + (int64_t)orow * p.ldg + tj * BN + c * 32 + c4) = make_uint4(o0, o1, o2, o3);
            }
            __syncwarp();
        }
    }
    if (diag) {
        const float rv = tc_ld_margin(t_row + (need_g ? BN : 0));
        const int row = ti * BM + warp * 32 + lane;
        if (row < p.sb) {
            p.r[row] = rv;
            if (p.s1_loss >= 0) {                   // this thread gathered this very row: its label is in a register
                p.z[row] = rv;
                p.u[row] = lprime_rt(p.s1_loss, rv, ylab);
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(256u) : "memory");
    }
    stamp_end(p.stamp);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *sym = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)sym;
    }
    return fn;
}

bool make_bf16_map(CUtensorMap *map, const void *base, uint64_t cols, uint64_t rows, uint64_t row_stride_elems,
                   uint32_t box_cols, uint32_t box_rows)
{
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    cuuint64_t dims[2] = {cols, rows};
    cuuint64_t strides[1] = {row_stride_elems * 2};
    cuuint32_t box[2] = {box_cols, box_rows};
    cuuint32_t estr[2] = {1, 1};
    return fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(base), dims, strides, box, estr,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

struct GramTcPlan {
    CUtensorMap tmY, tmX;
    int32_t n, rows_alloc;
};

// Y: [rows_alloc x ldy] BF16 (pad columns zero), xbf: [16 x ldxb] BF16 whose row 0 is the shadow and rows 1..15 zero.
GramTcPlan *gram_tc_plan_create(const uint16_t *Y, int32_t ldy, int32_t n, int32_t rows_alloc, const uint16_t *xbf,
                                int32_t ldxb, char *err, int errlen)
{
    GramTcPlan *pl = new GramTcPlan;
    pl->n = n;
    pl->rows_alloc = rows_alloc;
    // inner extent n: the K tail of the last 64-wide box is zero-filled by TMA
    if (!make_bf16_map(&pl->tmY, Y, (uint64_t)n, (uint64_t)rows_alloc, (uint64_t)ldy, BK, BM) ||
        !make_bf16_map(&pl->tmX, xbf, (uint64_t)n, (uint64_t)XR, (uint64_t)ldxb, BK, XR)) {
        snprintf(err, errlen, "cuTensorMapEncodeTiled failed (n = %d, ldy = %d, rows = %d)", n, ldy, rows_alloc);
        delete pl;
        return nullptr;
    }
    return pl;
}

void gram_tc_plan_destroy(GramTcPlan *p) { delete p; }

cudaError_t gram_tc_configure()
{
    cudaError_t e = cudaFuncSetAttribute(gram_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(gram_narrow_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kNwSmem);
}

int launch_gram_tc(cudaStream_t st, GramTcPlan *plan, int32_t row_base, int32_t sb, int32_t b, float *G, int32_t ldg, float *r,
                   int full_lower, int ksplit_opt, int num_sms, char *err, int errlen)
{
    GramParams p;
    p.G = G; p.r = r; p.ldg = ldg; p.sb = sb; p.b = b; p.n = plan->n; p.row_base = row_base; p.no_margin = r == nullptr;
    p.T = (sb + BM - 1) / BM;
    p.ntiles = p.T * (p.T + 1) / 2;
    p.kb_total = (plan->n + BK - 1) / BK;
    p.full_lower = full_lower;
    p.stamp = g_stamp;
    int ksplit = ksplit_opt;
    if (ksplit <= 0) {
        // fill the 148 SMs when there are few tiles -- but the cleared G, its memset node and the red.add epilogue
        // cost several microseconds, so only when a slice still holds >= 16 K blocks (1024 columns)
        ksplit = num_sms / p.ntiles;
        ksplit = std::min(ksplit, p.kb_total / 16);
        // ... and only when the split takes >= 24 K blocks off the critical path (measured: n = 2000, 32 K blocks:
        // splitting in 2 costs 3 us more than it saves; n = 4096, 64 K blocks: splitting in 4 saves 5 us)
        if (ksplit > 1 && p.kb_total - p.kb_total / ksplit < 24) ksplit = 1;
    }
    ksplit = std::max(1, std::min(ksplit, p.kb_total));
    p.ksplit = ksplit;
    int launches = 1;
    if (ksplit > 1) {
        // partial sums are added with red.global.add.f32: clear the rows of G and r this step writes
        cudaMemsetAsync(G, 0, sizeof(float) * (size_t)p.T * BM * ldg, st);
        if (r) cudaMemsetAsync(r, 0, sizeof(float) * (size_t)p.T * BM, st);
    }
    const int grid = std::min(p.ntiles * ksplit, num_sms);
    cudaError_t e = launch_pdl(gram_tc_kernel, dim3(grid), dim3(kThreads), kSmemBytes, st, 1, plan->tmY, plan->tmX, p);
    if (e != cudaSuccess) {
        snprintf(err, errlen, "gram_tc_kernel launch: %s", cudaGetErrorString(e));
        return -1;
    }
    return launches;
}

// Gather + Gram + margin in one kernel for n <= 64 (replaces launch_gather + launch_gram_tc for the step).
int launch_gram_narrow(cudaStream_t st, const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n,
                       const int32_t *idx, const StepParams *ind, int64_t idx_off, int32_t sb, int32_t b,
                       const uint16_t *xbf, int32_t ldxb, uint16_t *Y, int32_t ldy, float *yI, float *G, int32_t ldg,
                       float *r, int full_lower, int *err_flag, const S1Fuse *s1)
{
    NarrowParams p;
    p.A = A; p.lda = lda; p.m = m; p.y = y; p.idx = idx; p.ind = ind; p.idx_off = idx_off; p.xbf = xbf; p.ldxb = ldxb;
    p.Y = Y; p.yI = yI; p.G = G; p.r = r; p.err_flag = err_flag; p.ldy = ldy; p.ldg = ldg; p.sb = sb; p.b = b; p.n = n;
    p.T = (sb + BM - 1) / BM;
    p.full_lower = full_lower;
    p.s1_loss = s1 ? s1->loss : -1;
    p.z = s1 ? s1->z : nullptr;
    p.u = s1 ? s1->u : nullptr;
    p.stamp = g_stamp;
    const int tiles = p.T * (p.T + 1) / 2;
    return launch_pdl(gram_narrow_kernel, dim3(tiles), dim3(kNwThreads), kNwSmem, st, 1, p) == cudaSuccess ? 1 : -1;
}

}  // namespace casgd

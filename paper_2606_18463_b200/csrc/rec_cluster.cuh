// rec_cluster.cuh -- what the cluster kernels of the recurrence (recurrence_stream.cu, recurrence_chain.cu) share:
// cluster / mbarrier / st.async / cp.async wrappers, l' for the chain's critical path, and the two pieces of the outer
// iteration a recurrence cluster can absorb for small steps -- the margin r = Y x_hat of its rows before the chain
// (Alg. 1 line 3) and the update x <- x - alpha Y^T u after it (lines 16-17).
#pragma once
#include "common.cuh"

namespace casgd {

namespace {

constexpr int kRcThreads = 512, kRcWarps = 16;          // both kernels run 16 warps per CTA

__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t v;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(v));
    return v;
}
__device__ __forceinline__ uint32_t cluster_nctarank()
{
    uint32_t v;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(v));
    return v;
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t mapa_u32(uint32_t local_saddr, uint32_t cta)
{
    uint32_t remote;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(local_saddr), "r"(cta));
    return remote;
}
__device__ __forceinline__ void st_async_b32(uint32_t remote_addr, uint32_t value, uint32_t remote_bar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b32 [%0], %1, [%2];"
                 ::"r"(remote_addr), "r"(value), "r"(remote_bar) : "memory");
}
__device__ __forceinline__ void st_async_v4(uint32_t remote_addr, float v0, float v1, float v2, float v3, uint32_t remote_bar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.b32 [%0], {%1, %2, %3, %4}, [%5];"
                 ::"r"(remote_addr), "r"(__float_as_uint(v0)), "r"(__float_as_uint(v1)), "r"(__float_as_uint(v2)),
                   "r"(__float_as_uint(v3)), "r"(remote_bar) : "memory");
}
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
__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
// ... with an L2 eviction policy (createpolicy)
__device__ __forceinline__ void cp_async16_hint(uint32_t dst, const void *src, unsigned long long pol)
{
    asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "l"(pol) : "memory");
}
// evict_first for data read exactly once, else the default priority
__device__ __forceinline__ unsigned long long l2_policy(bool read_once)
{
    unsigned long long pol;
    if (read_once) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    else asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ float4 lds_f4(uint32_t saddr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(saddr));
    return v;
}

// Fused outer update for small steps (Alg. 1 lines 16-17): when a CTA's slice of Y is small (<= 136 KB, <= 2048 columns), g = Y^T u, x <- x - alpha g and the
// BF16 shadow are done by this kernel's cluster right after the chain -- every CTA already holds all of u in shared
// memory -- instead of by a fourth kernel: each CTA sums its slice of the rows, the per-CTA column sums meet in
// CTA 0's shared memory (distributed shared memory stores), and CTA 0 adds them in a fixed order and updates x.
struct FusedGrad {
    const uint16_t *Y;          // [sb x ldy] staged rows (null: no fusion)
    int32_t ldy, n;
    float *x_direct;
    const StepParams *ind;
    uint16_t *xbf;
    int32_t split_ld;
    float *r_fused;             // pipelined schedule, small Y: the margin of this CTA's rows is computed here (no margin kernel)
};
constexpr int kFgMaxLdy = 2048;                          // columns (padded) the fused update handles

// l' with the fast exponential and reciprocal on the chain's critical path where their error (~2^-21 relative)
// is far inside the tolerance on u; Poisson keeps the accurate expf (its error is amplified by e^z).
template <int LOSS>
__device__ __forceinline__ float lprime_chain(float z, float y)
{
    if (LOSS == CASGD_LOGISTIC) {
        const float t = y * z;
        const float e = __expf(-fabsf(t));               // in (0, 1]
        const float num = (t >= 0.f) ? e : 1.f;          // 1 / (1 + e^t) = num / (1 + e)
        return -y * __fdividef(num, 1.f + e);
    }
    return lprime<LOSS>(z, y);
}


// r = Y x_hat for `mine` rows of this CTA, row_of(t) giving the t-th one: LG lanes side by side on a row, four passes
// (row loads) in flight per lane. With CASGD_OPT_MARGIN_SPLIT the residue rows of the shadow are added (== FP32 x).
// The caller orders the stores before the readers (fence + barrier).
template <class RowOf>
__device__ __forceinline__ void fused_margin_rows(const FusedGrad &fg, int mine, RowOf row_of, int warp, int lane, int nwarps)
{
    const int nvec = fg.ldy >> 3;
    int LG = 1;
    while (LG < nvec && LG < 32) LG <<= 1;          // lanes side by side on a row; 32 / LG rows per warp and pass
    const int sub = lane % LG, rsub = lane / LG, RP = 32 / LG;
    // four passes at once: four row loads per lane in flight (a pass per L2 round trip was 3 us of prologue)
    for (int t0 = warp * RP * 4; t0 < mine; t0 += nwarps * RP * 4) {
        float acc[4] = {0.f, 0.f, 0.f, 0.f};
        const uint16_t *yr[4];
        bool on[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int t = t0 + q * RP + rsub;
            on[q] = t < mine;
            yr[q] = fg.Y + (int64_t)row_of(on[q] ? t : 0) * fg.ldy;
        }
        for (int cv = sub; cv < nvec; cv += LG) {
            uint4 v[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) v[q] = on[q] ? ld_dep_v4(yr[q] + cv * 8) : make_uint4(0u, 0u, 0u, 0u);
            const uint4 x0 = ld_dep_v4(fg.xbf + cv * 8);
#pragma unroll
            for (int q = 0; q < 4; ++q) acc[q] = dot8_bf16(v[q], x0, acc[q]);
            if (fg.split_ld) {
                const uint4 x1 = ld_dep_v4(fg.xbf + fg.split_ld + cv * 8), x2 = ld_dep_v4(fg.xbf + 2 * fg.split_ld + cv * 8);
#pragma unroll
                for (int q = 0; q < 4; ++q) acc[q] = dot8_bf16(v[q], x2, dot8_bf16(v[q], x1, acc[q]));
            }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            for (int o = LG >> 1; o > 0; o >>= 1) acc[q] += __shfl_xor_sync(0xffffffffu, acc[q], o);
            if (on[q] && sub == 0) fg.r_fused[row_of(t0 + q * RP + rsub)] = acc[q];
        }
    }
}

// g = Y^T u, x <- x - alpha g, shadow, by the whole cluster (every thread of every CTA calls this; u_loc = all of u in
// this CTA's shared memory; scratch = kRcThreads * 32 bytes, and C * ldy * 4 more in CTA 0).
__device__ __forceinline__ void fused_update_tail(const FusedGrad &fg, const float *u_loc, unsigned char *scratch, int s, int b,
                                          float alpha, int C, int crank)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int sb = s * b, ldy = fg.ldy;
    const int nvec = ldy >> 3;                      // 16-byte vectors per row (pad columns of Y are zero)
    int CV = 1;
    while (CV < nvec && CV < 64) CV <<= 1;          // threads side by side on a row
    const int RL = kRcThreads / CV;                   // rows in flight
    const int cvl = threadIdx.x % CV, rl = threadIdx.x / CV;
    const int rows_per_cta = (sb + C - 1) / C;
    const int r0 = crank * rows_per_cta, r1 = min(sb, r0 + rows_per_cta);
    float *red = reinterpret_cast<float *>(scratch);                     // [RL][CV * 8]
    float *gbuf = reinterpret_cast<float *>(scratch + kRcThreads * 8 * 4);   // CTA 0: [C][ldy]
    for (int cv0 = 0; cv0 < nvec; cv0 += CV) {      // (one pass unless ldy > 512)
        const int cv = cv0 + cvl;
        float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        if (cv < nvec) {
            for (int row = r0 + rl; row < r1; row += RL) {
                const uint4 v = ldg_nc_v4(fg.Y + (int64_t)row * ldy + cv * 8);
                const float uu = u_loc[row];
                acc[0] = fmaf(bf16lo(v.x), uu, acc[0]); acc[1] = fmaf(bf16hi(v.x), uu, acc[1]);
                acc[2] = fmaf(bf16lo(v.y), uu, acc[2]); acc[3] = fmaf(bf16hi(v.y), uu, acc[3]);
                acc[4] = fmaf(bf16lo(v.z), uu, acc[4]); acc[5] = fmaf(bf16hi(v.z), uu, acc[5]);
                acc[6] = fmaf(bf16lo(v.w), uu, acc[6]); acc[7] = fmaf(bf16hi(v.w), uu, acc[7]);
            }
        }
        // rows first meet inside a warp (lanes CV apart hold the same columns), then the 16 warps' sums in shared
        // memory: a serial sum over all RL row lanes by CV * 8 threads was half of this tail
        for (int o = CV; o < 32; o <<= 1)
#pragma unroll
            for (int e = 0; e < 8; ++e) acc[e] += __shfl_xor_sync(0xffffffffu, acc[e], o);
        const int groups = CV <= 32 ? kRcWarps : RL, gidx = CV <= 32 ? warp : rl;
        if (CV > 32 || lane < CV) {
#pragma unroll
            for (int e = 0; e < 8; ++e) red[gidx * (CV * 8) + cvl * 8 + e] = acc[e];
        }
        __syncthreads();
        // column sums of this CTA, in a fixed order, straight into CTA 0's gbuf[crank][col]
        const uint32_t gbuf0 = mapa_u32((uint32_t)__cvta_generic_to_shared(gbuf), 0u);
        for (int t = threadIdx.x; t < CV * 8; t += kRcThreads) {
            float sum = 0.f;
            for (int q = 0; q < groups; ++q) sum += red[q * (CV * 8) + t];
            const int col = cv0 * 8 + t;
            if (col < ldy)
                asm volatile("st.shared::cluster.f32 [%0], %1;" ::"r"(gbuf0 + 4u * (uint32_t)(crank * ldy + col)), "f"(sum) : "memory");
        }
        __syncthreads();
    }
    cluster_sync_all();                             // every CTA's sums are in CTA 0; nobody stores into a CTA any more
    if (crank == 0) {
        float *x = fg.ind ? fg.ind->x : fg.x_direct;
        for (int col = threadIdx.x; col < fg.n; col += kRcThreads) {
            float g = 0.f;
            for (int q = 0; q < C; ++q) g += gbuf[q * ldy + col];
            const float xn = fmaf(-alpha, g, x[col]);
            x[col] = xn;
            store_shadow(fg.xbf, fg.split_ld, col, xn);
        }
    }
}

}  // namespace

}  // namespace casgd

// recurrence_chain.cu -- the s-step inner residual correction, Alg. 1 lines 6-15, for SMALL blocks
// (b <= 64):   for j = 0..s-1:  z_j = r_j - alpha * sum_{k<j} G_{jk} u_k ;  u_j = l'(z_j, y_{I_j})      (all FP32, L236)
// with the dependent chain on ONE CTA.
//
// recurrence_stream.cu spreads the rows of every block over the 16 CTAs of a cluster, so each of the s - 1 hops of the
// chain crosses distributed shared memory: produce u_j -> st.async to 16 CTAs (~215 cycles) -> mbarrier wake-up -> next
// block. Measured 0.45-0.6 us per hop, and on the narrow-row workloads (SUSY-, epsilon-, poisson-shaped: b = 64, 32, 64)
// those hops ARE the outer iteration. Here the hop never leaves an SM:
//   chain CTA (rank 0)  owns all b rows of every block. Per hop it needs only the NEWEST W blocks of G's row block j
//       (b x W b floats, <= 32 KB: straight from L2 into registers, three hops ahead) and the older part of the sum as ONE
//       number per row: z_j = r_j - alpha (G_{j, j-W..j-1} u_{j-W..j-1} + P_j). 512/b lanes per row, a shuffle tree, l',
//       one __syncthreads. (Planned at ~400 cycles per hop; MEASURED 1100-1400, and the helpers pace the chain at
//       ~2600 -- slower than the streaming kernel, so this kernel is opt-in only: DESIGN.md section 6.)
//   helpers (ranks 1..15)  own rows h, h+15, ... of every block and form P_j[i] = sum_{k <= j-W-1} G_{ik} u_k: the whole
//       older part of the row, as soon as u_{j-W-1} has arrived
//       from the chain CTA, and st.async it into the chain CTA W+1 hops before it is needed -- both DSMEM crossings are
//       off the critical path.
// G's strict block-lower part is read exactly once (L180). The sum of a row is (window tree) + (helper tree): a fixed
// order, the same bits every run. For small steps the cluster then applies the outer update (rec_cluster.cuh).
#include "common.cuh"
#include "rec_cluster.cuh"

namespace casgd {

namespace {

constexpr int kCcCluster = 16;                          // 1 chain CTA + 15 helpers
constexpr int kCcMaxOwn = 5;                            // rows of a block one helper owns at most: ceil(64 / 15)
constexpr int kCcSmemCap = 227 * 1024;
constexpr int kCcPieces = 4;                            // 16-byte pieces of a hop's window one lane holds at most
constexpr int kCcMaxSb = 4096;                          // u and P live in shared memory

// Blocks of the chain CTA's window: it takes b * W b * 4 bytes per hop out of L2 (one SM pulls ~80 B/cycle, a hop
// is ~400 cycles), and W >= 2 is what the helpers' round trip needs.
__host__ __device__ inline int chain_window(int b)
{
    int w = 32768 / (4 * b * b);
    int tpr = 32;
    while (tpr * b > 512) tpr >>= 1;
    while (w * b > 4 * 4 * tpr) --w;                    // kCcPieces float4 per lane
    return w < 2 ? 0 : (w > 4 ? 4 : w);
}

struct ChainLayout {                    // byte offsets into dynamic shared memory; identical in both roles up to `ring`
    uint32_t u, p, ubar, pbar, red, ring, stage_bytes, depth, total;
};

__host__ __device__ inline ChainLayout chain_layout(int s, int b, bool helper)
{
    ChainLayout L;
    const int W = chain_window(b), H = kCcCluster - 1;
    uint32_t o = 0;
    L.u = o;     o += 4u * (uint32_t)(s * b);
    L.p = o;     o += 4u * (uint32_t)(s * b);
    o = (o + 7u) & ~7u;
    L.ubar = o;  o += 8u * (uint32_t)s;
    L.pbar = o;  o += 8u * (uint32_t)s;
    o = (o + 15u) & ~15u;
    L.red = o;   o += 2u * kRcWarps * 8u * 4u;          // helpers: [hop parity][warp][row]
    o = (o + 127u) & ~127u;
    L.ring = o;
    const int older = s - W - 1 > 1 ? s - W - 1 : 1;    // blocks of the longest older part
    const uint32_t bytes = helper ? (uint32_t)((b + H - 1) / H) * (uint32_t)older * (uint32_t)b * 4u
                                  : (uint32_t)b * (uint32_t)(W * b) * 4u;
    L.stage_bytes = (bytes + 127u) & ~127u;
    const uint32_t room = (uint32_t)kCcSmemCap > L.ring ? ((uint32_t)kCcSmemCap - L.ring) / L.stage_bytes : 0u;
    L.depth = room >= 4u ? 4u : (room >= 2u ? 2u : 0u);    // (cp.async.wait_group takes a constant)
    L.total = L.ring + L.depth * L.stage_bytes;
    return L;
}

__device__ __forceinline__ float4 ldg_nc_f4(const float *p)
{
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}
// one try of a barrier phase (no spinning: the result can be consumed later)
__device__ __forceinline__ uint32_t mbar_test(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok;
}
__device__ __forceinline__ float lds_f32(uint32_t saddr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(saddr));
    return v;
}
__device__ __forceinline__ void sts_f32(uint32_t saddr, float v)
{
    asm volatile("st.shared.f32 [%0], %1;" ::"r"(saddr), "f"(v) : "memory");
}
__device__ __forceinline__ float dot4(const float4 g, const float4 v, float acc)
{
    acc = fmaf(g.x, v.x, acc);
    acc = fmaf(g.y, v.y, acc);
    acc = fmaf(g.z, v.z, acc);
    return fmaf(g.w, v.w, acc);
}

#ifdef CASGD_CHAIN_TRACE
__device__ long long g_chain_trace[8192];
#define CT(i) do { if (tid == 0 && (i) < 8192) g_chain_trace[(i)] = clock64(); } while (0)
#else
#define CT(i) do { } while (0)
#endif

template <int LOSS>
__global__ void __launch_bounds__(kRcThreads, 1)
recurrence_chain_kernel(const float *G, int32_t ldg, const float *r, const float *yI, int32_t s, int32_t b, float alpha,
                        float *z, float *u, const FusedGrad fg, unsigned long long *stamp, int late_trigger)
{
    extern __shared__ __align__(128) unsigned char cc_smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int C = (int)cluster_nctarank(), crank = (int)cluster_ctarank();
    if (!late_trigger) pdl_trigger();                   // (see recurrence_stream.cu on the late trigger)
    const int W = chain_window(b), H = C - 1, sb = s * b;
    const bool helper = crank > 0;
    const ChainLayout L = chain_layout(s, b, helper);
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(cc_smem);
    const uint32_t us = base + L.u, ps = base + L.p, ubar = base + L.ubar, pbar = base + L.pbar;
    const uint32_t ring = base + L.ring, stage_bytes = L.stage_bytes;
    const int depth = (int)L.depth;

    const int h = crank - 1;                            // helper h owns rows h, h + H, ... of every block
    const int nown = helper && h < b ? (b - h + H - 1) / H : 0;
    for (int k = tid; k < s; k += kRcThreads) {
        mbar_init(ubar + 8u * k, 1);                    // helpers: block k of u from the chain CTA
        mbar_expect_tx(ubar + 8u * k, 4u * (uint32_t)b);
        mbar_init(pbar + 8u * k, 1);                    // chain CTA: the older part of block k's sums from the helpers
        mbar_expect_tx(pbar + 8u * k, 4u * (uint32_t)b);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    pdl_wait();                                         // G, r and y_I come from the Gram, margin and gather kernels
    stamp_begin(stamp);
    if (fg.r_fused) {
        // Alg. 1 line 3 folded in (small Y, pipelined schedule): row crank + t C is this CTA's t-th; the chain CTA reads
        // all of r after the cluster barrier below
        const int mine = crank < sb ? (sb - crank + C - 1) / C : 0;
        fused_margin_rows(fg, mine, [&](int t) { return crank + t * C; }, warp, lane, kRcWarps);
        __threadfence();
    }
    __syncthreads();                                    // the barriers exist before a thread of this CTA uses one

    if (!helper) {
        // ===================== chain CTA =====================
        int TPR = 32;                                   // lanes side by side on a row
        while (TPR * b > kRcThreads) TPR >>= 1;
        const int i = tid / TPR, sub = tid & (TPR - 1);
        const bool active = i < b, owner = active && sub == 0;
        // The window of a hop goes from L2 straight into REGISTERS, three hops ahead (lane (i, sub) holds pieces sub,
        // sub + TPR, ... of row i: at most kCcPieces float4). Two stagings through shared memory were measured first --
        // one cp.async.bulk per row (the lanes of a warp issue bulk copies one after the other, ~65 cycles each: 2100
        // cycles per hop) and 16-byte cp.async (the window's 32 KB in and out of shared memory, on the same pipe as the
        // u loads: 1400 cycles per hop) -- this one leaves shared memory to u alone.
        auto load = [&](int jj, float4 (&g)[kCcPieces]) {
            const int ncw = min(jj, W), nch = jj < s && active ? ncw * b >> 2 : 0;
            const float *src = G + (int64_t)(jj * b + i) * ldg + (jj - ncw) * b;
#pragma unroll
            for (int q = 0; q < kCcPieces; ++q) {
                const int c = sub + TPR * q;
                g[q] = c < nch ? ldg_nc_f4(src + 4 * c) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
        };
        float4 g0[kCcPieces], g1[kCcPieces], g2[kCcPieces], g3[kCcPieces];    // hops j, j+1, j+2, j+3
        load(0, g1); load(1, g2); load(2, g3);          // (hop 0 has no window: zeros)
        // u_j to the helpers: thread t < (b/4) H sends rows 4v .. 4v+3 to CTA dst as one 16-byte st.async
        const int nvec = b >> 2;
        const bool sender = tid < nvec * H;
        const int sv = tid % nvec, sdst = 1 + tid / nvec;
        const uint32_t s_loc = us + 16u * (uint32_t)sv;
        const uint32_t s_rem = mapa_u32(s_loc, (uint32_t)(sender ? sdst : 0)), s_bar = mapa_u32(ubar, (uint32_t)(sender ? sdst : 0));
        cluster_sync_all();                             // every CTA's barriers exist; r of the fused margin is complete
        float rr = 0.f, yy = 0.f;
        if (owner) { rr = ld_dep(r + i); yy = ld_dep(yI + i); }
        // running addresses: everything a hop touches moves by a constant, so the loop carries pointers, not products
        const int b4 = b >> 2, pstep = 4 * TPR;
        const int64_t rowstep = (int64_t)b * ldg;
        const float *srcl = G + (int64_t)(3 * b + i) * ldg + (3 > W ? (3 - W) * b : 0) + 4 * sub;    // hop 3, this lane's piece 0
        uint32_t uaddr = us + 16u * (uint32_t)sub;      // u of the window's first block, this lane's piece 0
        uint32_t paddr = ps + 4u * (uint32_t)i, pb = pbar, oaddr = us + 4u * (uint32_t)i;
        const float *rp = r + b + i, *yp = yI + b + i;
        float *zp = z + i, *up = u + i;
        uint32_t sl = s_loc, sr = s_rem, sb_ = s_bar;
#pragma unroll 1
        for (int j = 0; j < s; ++j) {
            float rn = 0.f, yn = 0.f;                   // r and y of the next hop, a hop ahead
            if (owner && j + 1 < s) { rn = ld_dep(rp); yn = ld_dep(yp); }
            CT(8 * j);
#pragma unroll
            for (int q = 0; q < kCcPieces; ++q) { g0[q] = g1[q]; g1[q] = g2[q]; g2[q] = g3[q]; }
            CT(8 * j + 1);
            {
                const int jl = j + 3;
                const int nchl = jl < s && active ? min(jl, W) * b4 : 0;
#pragma unroll
                for (int q = 0; q < kCcPieces; ++q)
                    g3[q] = sub + TPR * q < nchl ? ldg_nc_f4(srcl + q * pstep) : make_float4(0.f, 0.f, 0.f, 0.f);
                srcl += rowstep + (jl >= W ? b : 0);
            }
            CT(8 * j + 7);
            // the older blocks' part of this hop, from the helpers: asked for now, needed after the window's dot
            uint32_t p_ok = 1u;
            float pv = 0.f;
            const bool need_p = owner && j >= W + 1;
            if (need_p) p_ok = mbar_test(pb, 0u);
            float acc = 0.f;
            if (j > 0) {
                const int nch = active ? min(j, W) * b4 : 0;
                float4 uv[kCcPieces];
#pragma unroll
                for (int q = 0; q < kCcPieces; ++q)
                    uv[q] = sub + TPR * q < nch ? lds_f4(uaddr + 16u * (uint32_t)(TPR * q)) : make_float4(0.f, 0.f, 0.f, 0.f);
                const float a0 = dot4(g0[1], uv[1], dot4(g0[0], uv[0], 0.f));
                const float a1 = dot4(g0[3], uv[3], dot4(g0[2], uv[2], 0.f));
                acc = a0 + a1;
                for (int o = TPR >> 1; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
            }
            CT(8 * j + 2);
            if (owner) {
                if (need_p) {
                    while (!p_ok) p_ok = mbar_test(pb, 0u);
                    CT(8 * j + 3);
                    pv = lds_f32(paddr);
                }
                const float zz = fmaf(-alpha, acc + pv, rr);
                const float uu = lprime_chain<LOSS>(zz, yy);
                sts_f32(oaddr, uu);
                *zp = zz;
                *up = uu;
            }
            rr = rn; yy = yn;
            CT(8 * j + 4);
            __syncthreads();                            // u_j is complete
            CT(8 * j + 5);
            if (sender) {
                const float4 t = lds_f4(sl);
                st_async_v4(sr, t.x, t.y, t.z, t.w, sb_);
            }
            const uint32_t bb = 4u * (uint32_t)b;
            if (j >= W) uaddr += bb;
            paddr += bb; oaddr += bb; pb += 8u; sl += bb; sr += bb; sb_ += 8u;
            rp += b; yp += b; zp += b; up += b;
            CT(8 * j + 6);
        }
    } else {
        // ===================== helper =====================
        const int first = W + 1;                        // the first hop with an older part
        const int older = s - W - 1 > 1 ? s - W - 1 : 1;
        const uint32_t row_stride = 4u * (uint32_t)(older * b);
        // columns [0, (jj - W) b) of this helper's rows of block jj, lane-private pieces as in the chain CTA
        auto issue = [&](int jj) {
            if (jj < s) {
                const int nch = (jj - W) * b >> 2;
                const uint32_t dst = ring + (uint32_t)((jj - first) % depth) * stage_bytes;
                for (int a = 0; a < nown; ++a) {
                    const float *src = G + (int64_t)(jj * b + h + a * H) * ldg;
                    for (int c = tid; c < nch; c += kRcThreads) cp_async16(dst + (uint32_t)a * row_stride + 16u * c, src + 4 * c);
                }
            }
            cp_async_commit();
        };
#pragma unroll 1
        for (int jj = first; jj < first + depth - 1; ++jj) issue(jj);
        cluster_sync_all();
        float *red = reinterpret_cast<float *>(cc_smem + L.red);
        const uint32_t rem_ps = mapa_u32(ps, 0u), rem_pbar = mapa_u32(pbar, 0u);
        int ready = 0;                                  // blocks 0 .. ready-1 of u have arrived
        if (nown > 0) {
#pragma unroll 1
            for (int j = first; j < s; ++j) {
                const uint32_t st = (uint32_t)((j - first) % depth);
                issue(j + depth - 1);                   // into the stage this lane read a hop ago
                if (depth == 4) cp_async_wait<3>(); else cp_async_wait<1>();
                for (; ready <= j - W - 1; ++ready) mbar_wait(ubar + 8u * ready, 0u);
                const int nch = (j - W) * b >> 2;
                float acc[kCcMaxOwn];
#pragma unroll
                for (int a = 0; a < kCcMaxOwn; ++a) acc[a] = 0.f;
                const uint32_t srow = ring + st * stage_bytes;
#pragma unroll 1
                for (int c = tid; c < nch; c += kRcThreads) {
                    const float4 uv = lds_f4(us + 16u * c);
#pragma unroll
                    for (int a = 0; a < kCcMaxOwn; ++a)
                        if (a < nown) acc[a] = dot4(lds_f4(srow + (uint32_t)a * row_stride + 16u * c), uv, acc[a]);
                }
#pragma unroll
                for (int a = 0; a < kCcMaxOwn; ++a)
                    for (int o = 16; o > 0; o >>= 1) acc[a] += __shfl_xor_sync(0xffffffffu, acc[a], o);
                float *rb = red + (j & 1) * (kRcWarps * 8);
                if (lane == 0) {
#pragma unroll
                    for (int a = 0; a < kCcMaxOwn; ++a) rb[warp * 8 + a] = acc[a];
                }
                __syncthreads();
                if (warp < 3) {                         // 16 lanes per owned row add the warps' sums and send the total
                    const int a = tid >> 4, w = tid & 15;
                    float v = a < nown ? rb[w * 8 + a] : 0.f;
                    for (int o = 8; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                    if (w == 0 && a < nown)
                        st_async_b32(rem_ps + 4u * (uint32_t)(j * b + h + a * H), __float_as_uint(v), rem_pbar + 8u * j);
                }
            }
        }
    }

    cp_async_wait<0>();
    if (late_trigger) pdl_trigger();
    if (fg.Y) {
        // all of u is in every helper's shared memory once every block's barrier has completed; the chain CTA wrote it
        if (helper)
            for (int k = tid; k < s; k += kRcThreads) mbar_wait(ubar + 8u * k, 0u);
        __syncthreads();                                // ... and the rings are free: they become reduction buffers
        fused_update_tail(fg, reinterpret_cast<const float *>(cc_smem + L.u), cc_smem + L.ring, s, b, alpha, C, crank);
        __syncthreads();
        stamp_end(stamp);
        return;
    }
    __syncthreads();
    cluster_sync_all();                                 // no CTA leaves while others may still store into it
    stamp_end(stamp);
}

int chain_smem_bytes(int s, int b)
{
    const ChainLayout a = chain_layout(s, b, false), h = chain_layout(s, b, true);
    if (a.depth < 4 || h.depth < 2) return 0;          // (the chain CTA's ring is fixed at four stages)
    return (int)(a.total > h.total ? a.total : h.total);
}

template <int LOSS>
cudaError_t launch_chain(cudaStream_t st, const float *G, int32_t ldg, const float *r, const float *yI, int32_t s, int32_t b,
                         float alpha, float *z, float *u, const FusedGrad &fg, int late_trigger)
{
    const int smem = chain_smem_bytes(s, b);
    if (smem == 0) return cudaErrorInvalidConfiguration;
    return launch_pdl(recurrence_chain_kernel<LOSS>, dim3(kCcCluster), dim3(kRcThreads), (size_t)smem, st, kCcCluster, G, ldg, r, yI, s,
                      b, alpha, z, u, fg, g_stamp, late_trigger);
}

}  // namespace

cudaError_t recurrence_chain_configure()
{
    cudaError_t e = cudaSuccess;
    auto set = [&](auto kern) {
        if (e == cudaSuccess) e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kCcSmemCap);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    };
    set(recurrence_chain_kernel<CASGD_LOGISTIC>);
    set(recurrence_chain_kernel<CASGD_LINEAR>);
    set(recurrence_chain_kernel<CASGD_POISSON>);
    return e;
}

// Can the chain-CTA kernel run this shape? A cluster of 16, blocks of 8..64 rows (a window of >= 2 blocks within the
// chain CTA's L2 budget, <= 5 rows per helper), u and P within shared memory.
bool recurrence_chain_ok(int32_t s, int32_t b, int32_t ldg, int cluster)
{
    if (cluster < kCcCluster || s < 2 || b < 8 || b > 64 || b % 4 != 0 || ldg % 4 != 0 || s * b > kCcMaxSb) return false;
    if (chain_window(b) < 2 || (b + kCcCluster - 2) / (kCcCluster - 1) > kCcMaxOwn) return false;
    return chain_smem_bytes(s, b) > 0;
}

// Can it also do the outer update of this step (small Y)? Same rule as the streaming kernel's.
bool recurrence_chain_fuses_update(int32_t s, int32_t b, int32_t ldy)
{
    const ChainLayout a = chain_layout(s, b, false), h = chain_layout(s, b, true);
    const int64_t ring = std::min<int64_t>(a.total - a.ring, h.total - h.ring);
    const int64_t buffers = (int64_t)kRcThreads * 8 * 4 + (int64_t)kCcCluster * ldy * 4;
    return ldy <= kFgMaxLdy && (int64_t)s * b * ldy * 2 <= (int64_t)136 * 1024 * kCcCluster && buffers <= ring;
}

int launch_recurrence_chain(cudaStream_t st, const float *G, int32_t ldg, const float *r, const float *yI, int32_t s, int32_t b,
                            float alpha, int loss, float *z, float *u, const FusedUpdate *fu, int late_trigger)
{
    FusedGrad fg{};
    if (fu) fg = FusedGrad{fu->Y, fu->ldy, fu->n, fu->x, fu->ind, fu->xbf, fu->split_ld, fu->r_fused};
    cudaError_t e = loss == CASGD_LOGISTIC ? launch_chain<CASGD_LOGISTIC>(st, G, ldg, r, yI, s, b, alpha, z, u, fg, late_trigger)
                  : loss == CASGD_LINEAR  ? launch_chain<CASGD_LINEAR>(st, G, ldg, r, yI, s, b, alpha, z, u, fg, late_trigger)
                                          : launch_chain<CASGD_POISSON>(st, G, ldg, r, yI, s, b, alpha, z, u, fg, late_trigger);
    return e == cudaSuccess ? 1 : -1;
}

#ifdef CASGD_CHAIN_TRACE
extern "C" int casgd_chain_trace_dump(long long *dst_host, int n)
{
    cudaDeviceSynchronize();
    return (int)cudaMemcpyFromSymbol(dst_host, g_chain_trace, sizeof(long long) * (size_t)n);
}
#endif

}  // namespace casgd

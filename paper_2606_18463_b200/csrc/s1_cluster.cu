// s1_cluster.cu -- s = 1 (plain mini-batch SGD on BF16 rows with a BF16 shadow, PAPER.md:L99 with Recipe C's storage) for
// rows too wide for mini_step.cu's one CTA: ALL iterations of a call in one persistent launch of ONE thread-block cluster
// that splits the COLUMNS (the paper's own block-column idea, L141, across the SMs of a GPC instead of across GPUs).
//
// CTA c of C holds columns [c0, c1) of x in shared memory for the whole call and, per iteration,
//   gathers its column slice of the b sampled rows (Alg. 1 line 2; 16-byte cp.async, the next iteration's slice in flight),
//   forms the partial margins  p_c[i] = Y[i, c0:c1] . x_hat[c0:c1]  (line 3) and stores them into EVERY CTA of the cluster
//   (st.async into distributed shared memory, counted on the receiver's mbarrier) -- the one exchange of an iteration,
//   b floats per CTA pair -- and, once its own C * b partials have landed, adds them in rank order (every CTA gets the same bits), applies l' (lines 6-15 at
//   s = 1), and updates its own columns: x[c0:c1] -= alpha * Y[:, c0:c1]^T u (lines 16-17).
// No Gram, no recurrence, no global-memory round trip between the margin and the update, no kernel boundary per step:
// the kernel-per-stage path needs two launches and ~7-11 us per step here, and so does the FP32 baseline.
#include "common.cuh"
#include "rec_cluster.cuh"                  // lprime_chain

namespace casgd {

namespace {

constexpr int kScMaxThreads = 512, kScMaxWarps = 16;     // the launch picks 256 or 512 threads
constexpr int kScMaxB = 256;

struct S1Params {
    const uint16_t *A;
    int64_t lda, m;
    const float *y;
    const int32_t *idx;
    int64_t n_steps;
    int32_t n, ldy, b, exact_margin, cpc;     // cpc: columns per CTA (a multiple of 8)
    float alpha;
    float *x;
    uint16_t *xbf;
    int32_t ldxb, split;
    uint16_t *Y;                                    // exports of the last iteration
    float *yI, *r, *z, *u;
    int *err_flag;
    unsigned long long *stamp;
};

// two stages of the labels, the indices, the receive buffers and the Y slice: stage q at base + q * stride (scalars: an
// array of offsets indexed at run time lives in local memory)
struct S1Layout {
    uint32_t x, xm, u, yl, idx, vec_stride, recv, recv_stride, red, Y, Y_stride, total;
    int32_t lds;                                    // row stride of a Y slice in elements
};

__host__ __device__ inline S1Layout s1_layout(int b, int cpc, int C)
{
    S1Layout L;
    L.lds = cpc + 8;
    uint32_t o = 0;
    auto take = [&](uint32_t bytes) { const uint32_t at = o; o += (bytes + 15u) & ~15u; return at; };
    L.x = take(4u * cpc);
    L.xm = take(4u * cpc);                             // the margin's view of the slice: bf16-rounded, or x itself
    L.u = take(4u * b);
    L.vec_stride = (4u * b + 15u) & ~15u;
    L.yl = take(2u * L.vec_stride);
    L.idx = take(2u * L.vec_stride);
    L.recv_stride = (4u * (uint32_t)C * b + 15u) & ~15u;                     // [rank][row]
    L.recv = take(2u * L.recv_stride);
    L.red = take(4u * kScMaxWarps * cpc);
    L.Y_stride = (2u * (uint32_t)b * L.lds + 15u) & ~15u;
    L.Y = take(2u * L.Y_stride);
    L.total = o;
    return L;
}

__device__ __forceinline__ uint32_t sc_rank() { uint32_t v; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(v)); return v; }
__device__ __forceinline__ uint32_t sc_size() { uint32_t v; asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(v)); return v; }
__device__ __forceinline__ void sc_cluster_sync()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

// (one instantiation per loss, outer loops not unrolled, power-of-two lane groups: see mini_step.cu on code size)
// WIDE8: the margin takes eight rows per lane group (the launch checks that b and the slice width allow it; a kernel of its
// own so that the other shapes keep their smaller loop body)
template <int LOSS, bool WIDE8>
__global__ void __launch_bounds__(kScMaxThreads, 1)
s1_cluster_kernel(const S1Params p)
{
    extern __shared__ __align__(128) unsigned char sc_smem[];
    __shared__ __align__(8) unsigned long long sc_bars[2];       // one per receive buffer: C * b * 4 bytes complete a phase
    pdl_trigger();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthr = blockDim.x, nwarp = nthr >> 5;
    const int C = (int)sc_size(), crank = (int)sc_rank();
    const int b = p.b, n = p.n, cpc = p.cpc;
    const S1Layout L = s1_layout(b, cpc, C);
    const int lds = L.lds;
    const int c0 = crank * cpc;                          // first column of this CTA
    const int ncol = max(0, min(cpc, p.ldy - c0));       // columns of the (padded) row this CTA holds
    const int chunks = ncol >> 3;
    float *xs = reinterpret_cast<float *>(sc_smem + L.x);
    float *xm = reinterpret_cast<float *>(sc_smem + L.xm);
    float *us = reinterpret_cast<float *>(sc_smem + L.u);
    float *red = reinterpret_cast<float *>(sc_smem + L.red);
    const uint32_t smem0 = (uint32_t)__cvta_generic_to_shared(sc_smem);

#pragma unroll 1
    for (uint32_t o = L.Y + 16u * tid; o < L.total; o += 16u * nthr)
        *reinterpret_cast<uint4 *>(sc_smem + o) = make_uint4(0u, 0u, 0u, 0u);
    pdl_wait();
    stamp_begin(p.stamp);
#pragma unroll 1
    for (int k = tid; k < cpc; k += nthr) {
        const float t = c0 + k < n ? p.x[c0 + k] : 0.f;
        xs[k] = t;
        xm[k] = p.exact_margin ? t : __bfloat162float(__float2bfloat16_rn(t));
    }
    if (tid < b) {                                      // (b <= 256 = the threads: one index per thread and stage)
        reinterpret_cast<int32_t *>(sc_smem + L.idx)[tid] = p.idx[tid];
        if (p.n_steps > 1) reinterpret_cast<int32_t *>(sc_smem + L.idx + L.vec_stride)[tid] = p.idx[b + tid];
    }
    __syncthreads();

    int CH = 1, chs = 0;                                // gather, export: lanes side by side on a row slice (cpc <= 256: CH <= 32)
    while (CH < (cpc >> 3)) { CH <<= 1; ++chs; }
    const int csub = tid & (CH - 1), crow = tid >> chs, crows = nthr >> chs;

    auto issue_gather = [&](int64_t step) {
        const uint32_t q = (uint32_t)(step & 1);
        const int32_t *I = reinterpret_cast<const int32_t *>(sc_smem + L.idx + q * L.vec_stride);
        const uint32_t ybase = L.Y + q * L.Y_stride;
        if (csub < chunks) {
#pragma unroll 1
            for (int row = crow; row < b; row += crows) {
                const int64_t src = I[row];
                const uint32_t off = ybase + 2u * (uint32_t)(row * lds + csub * 8);
                if (src >= 0 && src < p.m)
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem0 + off), "l"(p.A + src * p.lda + c0 + csub * 8) : "memory");
                else *reinterpret_cast<uint4 *>(sc_smem + off) = make_uint4(0u, 0u, 0u, 0u);
            }
        }
        if (tid < b) {
            const int64_t src = I[tid];
            const uint32_t off = L.yl + q * L.vec_stride + 4u * (uint32_t)tid;
            if (src >= 0 && src < p.m) asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem0 + off), "l"(p.y + src) : "memory");
            else { *reinterpret_cast<float *>(sc_smem + off) = 0.f; if (crank == 0) flag_index_error(p.err_flag); }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    if (p.n_steps > 0) issue_gather(0);
    const uint32_t bar0 = (uint32_t)__cvta_generic_to_shared(sc_bars), rx_bytes = 4u * (uint32_t)(C * b);
    if (tid == 0) {
        mbar_init(bar0, 1); mbar_init(bar0 + 8u, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        mbar_expect_tx(bar0, rx_bytes); mbar_expect_tx(bar0 + 8u, rx_bytes);
    }
    sc_cluster_sync();                                  // every CTA's receive buffers and barriers exist before anyone stores

    int LG = 1, lgs = 0;
    while (LG < chunks && LG < 32) { LG <<= 1; ++lgs; }  // lanes side by side on a row slice
    const int rows_per_pass = nthr >> lgs, sub = tid & (LG - 1), mrow = tid >> lgs;
    const uint32_t recv_rank_off = 4u * (uint32_t)(crank * b);
    const bool wide8 = WIDE8 && LG >= 8;                 // (a last CTA with a narrower slice takes the plain path)

#pragma unroll 1
    for (int64_t step = 0; step < p.n_steps; ++step) {
        const uint32_t q = (uint32_t)(step & 1);
        const bool last = step + 1 == p.n_steps;
        if (!last) issue_gather(step + 1); else asm volatile("cp.async.commit_group;" ::: "memory");
        int32_t idx_next = 0;
        if (step + 2 < p.n_steps && tid < b) idx_next = p.idx[(step + 2) * b + tid];
        asm volatile("cp.async.wait_group 1;" ::: "memory");
        __syncthreads();
        uint16_t *Ys = reinterpret_cast<uint16_t *>(sc_smem + L.Y + q * L.Y_stride);
        const float *yl = reinterpret_cast<const float *>(sc_smem + L.yl + q * L.vec_stride);
        const uint32_t recv_q = L.recv + q * L.recv_stride;
        if ((n & 7) && c0 + ncol > n) {                 // the CTA that holds the row's last chunk: pad columns are zero
            if (tid < b)
                for (int c = n - c0; c < ncol; ++c) Ys[tid * lds + c] = 0;
            __syncthreads();
        }

        // ---- partial margins of this column slice, into every CTA's receive buffer
        if (WIDE8 && wide8) {
            // enough rows for every lane group to take EIGHT at once: the x chunk is read once per eight rows, and the eight
            // sums meet in one transposing reduction (7-9 shuffles for eight rows instead of 3-5 per row)
            const int o1 = LG >> 1, o2 = LG >> 2, o3 = LG >> 3;
            const bool u1 = sub & o1, u2 = sub & o2, u3 = sub & o3;
#pragma unroll 1
            for (int base = 0; base < b; base += rows_per_pass * 8) {
                const int i0 = base + mrow * 8;
                float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll 1
                for (int c = sub; c < chunks; c += LG) {
                    const float4 xa = *reinterpret_cast<const float4 *>(xm + c * 8), xb = *reinterpret_cast<const float4 *>(xm + c * 8 + 4);
#pragma unroll
                    for (int r8 = 0; r8 < 8; ++r8) {
                        if (i0 + r8 < b) {
                            const uint4 v = *reinterpret_cast<const uint4 *>(Ys + (i0 + r8) * lds + c * 8);
                            float a = acc[r8];
                            a = fmaf(bf16lo(v.x), xa.x, a); a = fmaf(bf16hi(v.x), xa.y, a);
                            a = fmaf(bf16lo(v.y), xa.z, a); a = fmaf(bf16hi(v.y), xa.w, a);
                            a = fmaf(bf16lo(v.z), xb.x, a); a = fmaf(bf16hi(v.z), xb.y, a);
                            a = fmaf(bf16lo(v.w), xb.z, a); a = fmaf(bf16hi(v.w), xb.w, a);
                            acc[r8] = a;
                        }
                    }
                }
                float t4[4], t2[2];
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    t4[k] = (u1 ? acc[k + 4] : acc[k]) + __shfl_xor_sync(0xffffffffu, u1 ? acc[k] : acc[k + 4], o1);
#pragma unroll
                for (int k = 0; k < 2; ++k)
                    t2[k] = (u2 ? t4[k + 2] : t4[k]) + __shfl_xor_sync(0xffffffffu, u2 ? t4[k] : t4[k + 2], o2);
                float tot = (u3 ? t2[1] : t2[0]) + __shfl_xor_sync(0xffffffffu, u3 ? t2[0] : t2[1], o3);
                for (int o = o3 >> 1; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
                // this lane now holds the sum of row i0 + (u1 u2 u3); the o3 lanes of a row share its C remote stores
                const int i = i0 + (u1 ? 4 : 0) + (u2 ? 2 : 0) + (u3 ? 1 : 0);
                if (i < b)
#pragma unroll 1
                    for (int dstc = sub & (o3 - 1); dstc < C; dstc += o3) {
                        const uint32_t remote = mapa_u32(smem0 + recv_q + recv_rank_off + 4u * (uint32_t)i, (uint32_t)dstc);
                        st_async_b32(remote, __float_as_uint(tot), mapa_u32(bar0 + 8u * q, (uint32_t)dstc));
                    }
            }
        } else
#pragma unroll 1
        for (int i0 = 0; i0 < b; i0 += rows_per_pass) {
            const int i = i0 + mrow;
            float acc = 0.f, acc2 = 0.f;
#pragma unroll 1
            for (int c = sub; c < chunks && i < b; c += LG) {
                const uint4 v = *reinterpret_cast<const uint4 *>(Ys + i * lds + c * 8);
                const float4 xa = *reinterpret_cast<const float4 *>(xm + c * 8), xb = *reinterpret_cast<const float4 *>(xm + c * 8 + 4);
                acc = fmaf(bf16lo(v.x), xa.x, acc); acc2 = fmaf(bf16hi(v.x), xa.y, acc2);
                acc = fmaf(bf16lo(v.y), xa.z, acc); acc2 = fmaf(bf16hi(v.y), xa.w, acc2);
                acc = fmaf(bf16lo(v.z), xb.x, acc); acc2 = fmaf(bf16hi(v.z), xb.y, acc2);
                acc = fmaf(bf16lo(v.w), xb.z, acc); acc2 = fmaf(bf16hi(v.w), xb.w, acc2);
            }
            acc += acc2;
            for (int o = LG >> 1; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
            // lane `sub` of the row's group stores to CTA sub, sub + LG, ...: the C remote stores of a row are spread over its lanes
            if (i < b)
#pragma unroll 1
                for (int dstc = sub; dstc < C; dstc += LG) {
                    uint32_t remote;
                    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(smem0 + recv_q + recv_rank_off + 4u * (uint32_t)i), "r"((uint32_t)dstc));
                    st_async_b32(remote, __float_as_uint(acc), mapa_u32(bar0 + 8u * q, (uint32_t)dstc));
                }
        }
        // all C * b partials of this iteration have landed HERE (st.async counts them on this buffer's barrier): no
        // cluster-wide barrier per iteration -- a CTA can be at most one iteration ahead of the slowest (it needs
        // everybody's partials to go on), which is what the two receive buffers allow
        mbar_wait(bar0 + 8u * q, (uint32_t)(step >> 1) & 1u);

        // ---- r = sum over ranks (rank order: identical bits in every CTA), u = l'(r, y_I)
        const float *rv = reinterpret_cast<const float *>(sc_smem + recv_q);
        if (tid < b) {
            const int i = tid;
            float rr = 0.f;
#pragma unroll 4
            for (int k = 0; k < C; ++k) rr += rv[k * b + i];
            const float uu = lprime_chain<LOSS>(rr, yl[i]);
            us[i] = uu;
            if (last && crank == 0) { p.yI[i] = yl[i]; p.r[i] = rr; p.z[i] = rr; p.u[i] = uu; }
        }
        __syncthreads();
        if (tid == 0) mbar_expect_tx(bar0 + 8u * q, rx_bytes);      // this buffer's next phase (iteration step + 2), armed
                                                                    // before this CTA's partials of step + 1 let anyone get there

        // ---- update of this CTA's columns: CH lanes side by side on a row slice (8 columns each), the rows dealt over
        // the lane groups; the groups of a warp meet by shuffles, the warps through shared memory
        {
            float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
            if (csub < chunks)
#pragma unroll 2
                for (int i = crow; i < b; i += crows) {
                    const uint4 v = *reinterpret_cast<const uint4 *>(Ys + i * lds + csub * 8);
                    const float uu = us[i];
                    acc[0] = fmaf(bf16lo(v.x), uu, acc[0]); acc[1] = fmaf(bf16hi(v.x), uu, acc[1]);
                    acc[2] = fmaf(bf16lo(v.y), uu, acc[2]); acc[3] = fmaf(bf16hi(v.y), uu, acc[3]);
                    acc[4] = fmaf(bf16lo(v.z), uu, acc[4]); acc[5] = fmaf(bf16hi(v.z), uu, acc[5]);
                    acc[6] = fmaf(bf16lo(v.w), uu, acc[6]); acc[7] = fmaf(bf16hi(v.w), uu, acc[7]);
                }
#pragma unroll 1
            for (int o = CH; o < 32; o <<= 1)
#pragma unroll
                for (int e = 0; e < 8; ++e) acc[e] += __shfl_xor_sync(0xffffffffu, acc[e], o);
            if (csub < chunks && lane < CH) {
#pragma unroll
                for (int e = 0; e < 8; ++e) red[warp * cpc + csub * 8 + e] = acc[e];
            }
        }
        __syncthreads();
#pragma unroll 1
        for (int k = tid; k < ncol; k += nthr) {
            float g = 0.f;
#pragma unroll 8
            for (int w = 0; w < nwarp; ++w) g += red[w * cpc + k];
            const float xn = fmaf(-p.alpha, g, xs[k]);
            xs[k] = xn;
            xm[k] = p.exact_margin ? xn : __bfloat162float(__float2bfloat16_rn(xn));
        }
        if (last && csub < chunks)
#pragma unroll 1
            for (int row = crow; row < b; row += crows)
                *reinterpret_cast<uint4 *>(p.Y + (int64_t)row * p.ldy + c0 + csub * 8) = *reinterpret_cast<const uint4 *>(Ys + row * lds + csub * 8);
        if (step + 2 < p.n_steps && tid < b) reinterpret_cast<int32_t *>(sc_smem + L.idx + q * L.vec_stride)[tid] = idx_next;
        __syncthreads();
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
#pragma unroll 1
    for (int k = tid; k < ncol; k += nthr)
        if (c0 + k < n) {
            p.x[c0 + k] = xs[k];
            store_shadow(p.xbf, p.split ? p.ldxb : 0, c0 + k, xs[k]);
        }
    sc_cluster_sync();                                  // no CTA leaves while another may still store into it
    stamp_end(p.stamp);
}

constexpr int kScSmemCap = 200 * 1024;

// cluster size and columns per CTA for a row of ldy (padded) columns
void s1_cluster_shape(int32_t ldy, int *C, int *cpc)
{
    int c = ldy >= 16 * 64 ? 16 : 8;
    int per = ((ldy + c - 1) / c + 7) & ~7;
    *C = c;
    *cpc = per;
}

}  // namespace

cudaError_t s1_cluster_configure()
{
    cudaError_t e = cudaSuccess;
    auto set = [&](auto *k) {
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, kScSmemCap);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    };
    set(s1_cluster_kernel<CASGD_LOGISTIC, false>); set(s1_cluster_kernel<CASGD_LOGISTIC, true>);
    set(s1_cluster_kernel<CASGD_LINEAR, false>);   set(s1_cluster_kernel<CASGD_LINEAR, true>);
    set(s1_cluster_kernel<CASGD_POISSON, false>);  set(s1_cluster_kernel<CASGD_POISSON, true>);
    return e;
}

// s = 1, rows of >= 128 bytes (8 columns per CTA), b <= 256, everything of a CTA within its shared memory. Measured against
// mini_step.cu's one CTA (us per iteration): n = 64, b = 128: 1.96 against 2.27; n = 128, b = 128: 2.16 against 3.98;
// n = 248, b = 64: 1.93 against 5.31 -- and the other way round only for steps of <= 4 KB (n = 64, b = 16: 1.52 against 1.19)
bool s1_cluster_ok(int32_t n, int32_t ldy, int32_t b, int cluster_max)
{
    if (ldy != ((n + 7) & ~7) || ldy * 2 < 128 || b < 1 || b > kScMaxB) return false;
    int C, cpc;
    s1_cluster_shape(ldy, &C, &cpc);
    if (C > cluster_max) return false;
    return s1_layout(b, cpc, C).total <= (uint32_t)kScSmemCap;
}

int launch_s1_cluster(cudaStream_t st, const uint16_t *A, int64_t lda, const float *y, int64_t m, int32_t n, int32_t ldy,
                      const int32_t *idx, int64_t n_steps, int32_t b, float alpha, int loss, int exact_margin, float *x,
                      uint16_t *xbf, int32_t ldxb, int split, uint16_t *Y, float *yI, float *r, float *z, float *u, int *err_flag)
{
    S1Params p;
    int C;
    s1_cluster_shape(ldy, &C, &p.cpc);
    p.A = A; p.lda = lda; p.m = m; p.y = y; p.idx = idx; p.n_steps = n_steps; p.n = n; p.ldy = ldy; p.b = b;
    p.exact_margin = exact_margin; p.alpha = alpha; p.x = x; p.xbf = xbf; p.ldxb = ldxb; p.split = split;
    p.Y = Y; p.yI = yI; p.r = r; p.z = z; p.u = u; p.err_flag = err_flag; p.stamp = g_stamp;
    const S1Layout L = s1_layout(b, p.cpc, C);
    // measured: 16 warps per CTA pay once a CTA's slice of a step is tens of KB (n = 4096, b = 128: 6.7 against 7.7 us);
    // below that the barriers of 8 warps are cheaper (n = 2000, b = 32: 1.96 against 2.13)
    const int threads = (int64_t)b * p.cpc * 2 >= (32 << 10) ? kScMaxThreads : 256;
    // eight rows per lane group in the margin: when every group of LG lanes (LG = the slice's 16-byte pieces rounded up to
    // a power of two, 8..32) gets eight rows
    int LG = 1;
    while (LG < p.cpc / 8 && LG < 32) LG <<= 1;
    const bool wide8 = LG >= 8 && b >= 8 * (threads / LG);
    auto pick = [&](auto *narrow, auto *wide) { return wide8 ? wide : narrow; };
    auto *kern = loss == CASGD_LOGISTIC ? pick(s1_cluster_kernel<CASGD_LOGISTIC, false>, s1_cluster_kernel<CASGD_LOGISTIC, true>)
               : loss == CASGD_LINEAR  ? pick(s1_cluster_kernel<CASGD_LINEAR, false>, s1_cluster_kernel<CASGD_LINEAR, true>)
                                       : pick(s1_cluster_kernel<CASGD_POISSON, false>, s1_cluster_kernel<CASGD_POISSON, true>);
    return launch_pdl(kern, dim3(C), dim3(threads), (size_t)L.total, st, C, p) == cudaSuccess ? 1 : -1;
}

}  // namespace casgd

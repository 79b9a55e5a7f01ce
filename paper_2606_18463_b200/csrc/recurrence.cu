// recurrence.cu -- the s-step inner residual correction, Alg. 1 lines 6-15:
//   for j = 0..s-1:  z_j = r_j - alpha * sum_{k<j} G_{jk} u_k ;  u_j = l'(z_j, y_{I_j})
// All FP32 (the paper requires u_c = u_sigma = FP32: L236, Table 3). Only blocks k < j of G are read
// ("strict block-lower", L180). The chain is serial in j; inside a step the b rows and the j*b-long
// dot products are parallel.
//
// Two kernels:
//   recurrence_cta_kernel   one CTA, u in shared memory, __syncthreads per step. For small G_L.
//   recurrence_grid_kernel  all SMs (cooperative launch, one CTA per SM). Each warp owns a few rows of G
//       (row i -> warp i mod W, so the b rows of a block sit on b different SMs) and keeps one lane-partial
//       dot product per row in registers. u_k travels between SMs as 8-byte {value, tag} words through L2
//       (the tag is a per-launch epoch, so a word is valid the moment it is visible: no flag, no fence,
//       one L2 round trip per step). When u_k lands every warp adds G[row, block k] . u_k to its rows
//       (the G loads are issued BEFORE the poll, so they are in flight while it spins), and the warps that own
//       rows of block k+1 reduce, apply l', and publish. The whole strict block-lower G is read exactly once,
//       by 148 SMs in parallel, instead of through one SM.
#include <cuda/atomic>

#include "common.cuh"

namespace casgd {

// ---------------------------------------------------------------------------- one CTA ---

template <int LOSS>
__global__ void __launch_bounds__(1024)
recurrence_cta_kernel(const float *G, int32_t ldg, const float *r, const float *yI,
                      int32_t s, int32_t b, float alpha, float *z, float *u, unsigned long long *stamp)
{
    extern __shared__ float u_s[];                    // [s*b]
    pdl_trigger();
    pdl_wait();
    stamp_begin(stamp);
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
    stamp_end(stamp);
}

// --------------------------------------------------------------------------- all SMs ---

constexpr int kRecThreads = 256;
constexpr int kRecWarps = kRecThreads / 32;

__device__ __forceinline__ void st_tagged(unsigned long long *p, float v, uint32_t tag)
{
    const unsigned long long w = ((unsigned long long)tag << 32) | (unsigned long long)__float_as_uint(v);
    asm volatile("st.relaxed.gpu.global.b64 [%0], %1;" ::"l"(p), "l"(w) : "memory");
}
__device__ __forceinline__ void ld_tagged_x4(const unsigned long long *p, uint32_t (&v)[4], uint32_t (&t)[4])
{
    // two 16-byte volatile loads: {v0, t0, v1, t1}, {v2, t2, v3, t3}; each 8-byte word was written whole
    asm volatile("ld.volatile.global.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v[0]), "=r"(t[0]), "=r"(v[1]), "=r"(t[1]) : "l"(p) : "memory");
    asm volatile("ld.volatile.global.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v[2]), "=r"(t[2]), "=r"(v[3]), "=r"(t[3]) : "l"(p + 2) : "memory");
}
__device__ __forceinline__ void ld_tagged_x1(const unsigned long long *p, uint32_t &v, uint32_t &t)
{
    asm volatile("ld.volatile.global.v2.u32 {%0, %1}, [%2];" : "=r"(v), "=r"(t) : "l"(p) : "memory");
}

// VEC: b % 4 == 0, so block-column offsets k*b are 16-byte aligned in G (ldg % 4 == 0) and in shared memory;
// each lane takes 4 consecutive columns per 128-column chunk. Otherwise one column per lane per 32-column
// chunk. MAXR bounds the rows one warp owns (ceil(sb / W)).
// Polling: every SM spinning on the same 8 b bytes would queue on the one or two L2 slices that hold them
// (measured: 5.8 us per step with 1184 polling warps). So (a) a CTA polls each word once -- thread c takes
// column c and drops the value into shared memory, one __syncthreads, then all warps read it there -- and
// (b) the producer writes `nrep` replicas 128 KB apart and CTA i polls replica i mod nrep.
template <int LOSS, int MAXR, bool VEC>
__global__ void __launch_bounds__(kRecThreads, 1)
recurrence_grid_kernel(const float *G, int32_t ldg, const float *r,
                       const float *yI, int32_t s, int32_t b, float alpha, float *z,
                       float *u, unsigned long long *utag, int32_t nrep,
                       unsigned *epoch, unsigned *done, unsigned long long *stamp)
{
    extern __shared__ __align__(16) float u_s[];        // [s*b]: u as it arrives
    __shared__ int s_last;
    stamp_begin(stamp);
    const uint32_t tag = *reinterpret_cast<volatile unsigned *>(epoch);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int W = gridDim.x * kRecWarps;
    const int gw = warp * gridDim.x + blockIdx.x;       // consecutive rows sit on different SMs
    const int sb = s * b;
    const int R = gw < sb ? (sb - 1 - gw) / W + 1 : 0;  // rows gw, gw + W, ..., gw + (R-1) W
    const unsigned long long *my_rep = utag + (size_t)(blockIdx.x % nrep) * CASGD_MAX_SB;

    float acc[MAXR], rv[MAXR], yv[MAXR];
    int blk[MAXR];
#pragma unroll
    for (int t = 0; t < MAXR; ++t) {
        acc[t] = 0.f;
        const int row = gw + t * W;
        const bool own = t < R;
        rv[t] = own ? ld_dep(r + row) : 0.f;
        yv[t] = own ? ld_dep(yI + row) : 0.f;
        blk[t] = own ? row / b : -1;
    }
    int last_blk = -1;
#pragma unroll
    for (int t = 0; t < MAXR; ++t) last_blk = max(last_blk, blk[t]);
    if (threadIdx.x == 0) s_last = -1;
    __syncthreads();
    if (lane == 0) atomicMax(&s_last, last_blk);
    __syncthreads();
    const int cta_last = s_last;                        // this CTA needs u_0 .. u_{cta_last - 1}

    auto finalize = [&](int t, int row) {
        const float a = warp_sum(acc[t]);               // every lane holds the sum
        const float zz = fmaf(-alpha, a, rv[t]);
        const float uu = lprime<LOSS>(zz, yv[t]);
        if (lane < nrep) st_tagged(utag + (size_t)lane * CASGD_MAX_SB + row, uu, tag);   // what the other SMs wait for
        if (lane == 0) {
            z[row] = zz;
            u[row] = uu;
        }
    };

    // rows of block 0 depend on nothing
#pragma unroll
    for (int t = 0; t < MAXR; ++t)
        if (blk[t] == 0) finalize(t, gw + t * W);

    constexpr int CW = VEC ? 128 : 32;                  // columns per chunk
    for (int k = 0; k < cta_last; ++k) {                // consume u_k; rows of blocks > k need it
        const int c_first = VEC ? lane * 4 : lane;
        const int64_t col0 = (int64_t)k * b;
        // chunk 0 of G for this warp's rows: in flight while the CTA waits for u_k
        float4 g4[VEC ? MAXR : 1];
        float g1[VEC ? 1 : MAXR];
#pragma unroll
        for (int t = 0; t < MAXR; ++t) {
            const bool need = blk[t] > k && c_first < b;
            const float *gp = G + (int64_t)(gw + t * W) * ldg + col0 + c_first;
            if (VEC) {
                g4[t] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (need) {
                    const uint4 w = ldg_nc_v4(gp);
                    g4[t] = make_float4(__uint_as_float(w.x), __uint_as_float(w.y), __uint_as_float(w.z),
                                        __uint_as_float(w.w));
                }
            } else {
                g1[t] = need ? __ldcg(gp) : 0.f;
            }
        }
        // the CTA's one poll of u_k
        for (int c = threadIdx.x; c < b; c += kRecThreads) {
            uint32_t v, tg;
            do { ld_tagged_x1(my_rep + col0 + c, v, tg); } while (tg != tag);
            u_s[col0 + c] = __uint_as_float(v);
        }
        __syncthreads();
        if (k < last_blk) {
            if (VEC) {
                if (c_first < b) {
                    const float4 uv = *reinterpret_cast<const float4 *>(u_s + col0 + c_first);
#pragma unroll
                    for (int t = 0; t < MAXR; ++t) {
                        acc[t] = fmaf(g4[t].x, uv.x, acc[t]);
                        acc[t] = fmaf(g4[t].y, uv.y, acc[t]);
                        acc[t] = fmaf(g4[t].z, uv.z, acc[t]);
                        acc[t] = fmaf(g4[t].w, uv.w, acc[t]);
                    }
                }
            } else {
                const float uv = c_first < b ? u_s[col0 + c_first] : 0.f;
#pragma unroll
                for (int t = 0; t < MAXR; ++t) acc[t] = fmaf(g1[t], uv, acc[t]);
            }
            // wide blocks: the remaining chunks
            for (int c = CW + c_first; c < b; c += CW) {
#pragma unroll
                for (int t = 0; t < MAXR; ++t) {
                    if (blk[t] <= k) continue;
                    const float *gp = G + (int64_t)(gw + t * W) * ldg + col0 + c;
                    if (VEC) {
                        const uint4 w = ldg_nc_v4(gp);
                        const float4 uv = *reinterpret_cast<const float4 *>(u_s + col0 + c);
                        acc[t] = fmaf(__uint_as_float(w.x), uv.x, acc[t]);
                        acc[t] = fmaf(__uint_as_float(w.y), uv.y, acc[t]);
                        acc[t] = fmaf(__uint_as_float(w.z), uv.z, acc[t]);
                        acc[t] = fmaf(__uint_as_float(w.w), uv.w, acc[t]);
                    } else {
                        acc[t] = fmaf(__ldcg(gp), u_s[col0 + c], acc[t]);
                    }
                }
            }
#pragma unroll
            for (int t = 0; t < MAXR; ++t)
                if (blk[t] == k + 1) finalize(t, gw + t * W);
        }
    }

    // the last CTA to finish retires the epoch, which invalidates every tagged word at once
    __syncthreads();
    if (threadIdx.x == 0) {
        cuda::atomic_ref<unsigned, cuda::thread_scope_device> d(*done);
        if (d.fetch_add(1u, cuda::memory_order_acq_rel) == gridDim.x - 1) {
            d.store(0u, cuda::memory_order_relaxed);
            *epoch = (tag + 1u == 0u) ? 1u : tag + 1u;  // 0 is the value of never-written words
        }
    }
    stamp_end(stamp);
}

// --------------------------------------------------------------- one thread-block cluster ---
// The chain of s-1 dependent steps is bound by how fast u_k gets from the SMs that produce it to the SMs that
// need it. Through L2 that hop costs ~1.5 us (measured above); between the CTAs of one cluster it is a remote
// shared-memory store (~0.1 us). So: one cluster of C (16, else 8) CTAs runs the whole recurrence.
//   * Every CTA holds all of u in its own shared memory, plus one mbarrier per block k that expects 4b bytes.
//     A finished u value goes to all C copies with st.async (...mbarrier::complete_tx::bytes): the store and
//     the barrier's byte count travel together, so consumers sleep in mbarrier.try_wait instead of hammering
//     shared memory, and a block is usable the moment its last value lands.
//   * Left-looking: at step j the b rows of block j are dealt to the CTAs (row q -> CTA q mod C); inside a CTA a
//     row belongs to one warp or, when there are fewer rows than warps, to several warps that split its
//     128-column chunks and hand their partial sums to the row's lead warp through shared memory. Each warp
//     walks its columns oldest first, so only the newest block is ever waited for.
//   * Steps alternate between two groups of warps (even j / odd j): while one group waits for the newest u,
//     the other is already streaming the older columns of the next step, which hides the L2 latency of G.
// G streams from L2 (where the Gram kernel just left it) with 4 x 16-byte loads in flight per lane.
// Needs b % 4 == 0 (16-byte loads at block-column offsets).

constexpr int kChainThreads = 512;
constexpr int kChainWarps = kChainThreads / 32;
constexpr int kChainGroups = 2;
constexpr int kGroupWarps = kChainWarps / kChainGroups;
constexpr int kChainUnroll = 4;

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
__device__ __forceinline__ void chain_bar_wait(uint32_t bar)
{
    uint32_t ok;
    do {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\nselp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(bar) : "memory");
    } while (!ok);
}

template <int LOSS>
__global__ void __launch_bounds__(kChainThreads, 1)
recurrence_cluster_kernel(const float *G, int32_t ldg, const float *r,
                          const float *yI, int32_t s, int32_t b, float alpha, float *z,
                          float *u, unsigned long long *stamp)
{
    extern __shared__ __align__(16) unsigned char chain_smem[];    // u_s[s*b] floats, then bars[s]
    __shared__ volatile float part[2][kChainWarps];
    __shared__ volatile int pflag[2][kChainWarps];                 // step whose partial sits in part[.][w]
    __shared__ volatile int cons[kChainWarps];                     // last step whose partial the lead has read
    pdl_trigger();
    pdl_wait();
    stamp_begin(stamp);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int C = (int)cluster_nctarank(), crank = (int)cluster_ctarank();
    const int sb = s * b;
    float *u_s = reinterpret_cast<float *>(chain_smem);
    const uint32_t us_base = (uint32_t)__cvta_generic_to_shared(u_s);
    const uint32_t bar_base = us_base + 4u * (uint32_t)sb;         // sb % 4 == 0: 8-byte aligned
    for (int k = threadIdx.x; k < s; k += kChainThreads) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_base + 8u * k) : "memory");
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_base + 8u * k), "r"(4u * b) : "memory");
    }
    if (threadIdx.x < kChainWarps) {
        pflag[0][threadIdx.x] = -1;
        pflag[1][threadIdx.x] = -1;
        cons[threadIdx.x] = -1;
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();
    cluster_sync_all();                                 // nobody signals a barrier that is not initialised yet

    int ready = 0;                                      // blocks 0 .. ready-1 of u are complete in u_s (this warp's view)

    // dot of row `row` with u over the 128-column chunks e = first, first + stride, ... counted from the END of
    // [0, L) (e = 0 is the newest chunk), walked oldest first
    auto dot_chunks = [&](int row, int L, int first, int stride) -> float {
        const int nchunks = (L + 127) >> 7;
        float acc = 0.f;
        if (first >= nchunks) return acc;
        const float *g = G + (int64_t)row * ldg + lane * 4;
        int e = first + ((nchunks - 1 - first) / stride) * stride;          // the oldest of this warp's chunks
        for (; e >= first; e -= kChainUnroll * stride) {
            uint4 gv[kChainUnroll];
#pragma unroll
            for (int q = 0; q < kChainUnroll; ++q) {
                const int eq = e - q * stride;
                const int col = (nchunks - 1 - eq) * 128 + lane * 4;
                gv[q] = make_uint4(0u, 0u, 0u, 0u);
                if (eq >= first && col < L) gv[q] = ldg_nc_v4(g + (nchunks - 1 - eq) * 128);
            }
#pragma unroll
            for (int q = 0; q < kChainUnroll; ++q) {
                const int eq = e - q * stride;
                if (eq >= first) {                                          // warp-uniform
                    const int c0 = (nchunks - 1 - eq) * 128;
                    const int need = (min(c0 + 128, L) - 1) / b;            // newest block this chunk touches
                    while (ready <= need) { chain_bar_wait(bar_base + 8u * ready); ++ready; }
                    const int col = c0 + lane * 4;
                    if (col < L) {
                        const float4 uv = *reinterpret_cast<const float4 *>(u_s + col);
                        acc = fmaf(__uint_as_float(gv[q].x), uv.x, acc);
                        acc = fmaf(__uint_as_float(gv[q].y), uv.y, acc);
                        acc = fmaf(__uint_as_float(gv[q].z), uv.z, acc);
                        acc = fmaf(__uint_as_float(gv[q].w), uv.w, acc);
                    }
                }
            }
        }
        return acc;
    };

    auto publish = [&](int j, int row, float total, float rr, float yy) {
        const float zz = fmaf(-alpha, total, rr);
        const float uu = lprime<LOSS>(zz, yy);
        if (lane < C && j + 1 < s)
            st_async_b32(mapa_u32(us_base + 4u * (uint32_t)row, (uint32_t)lane), __float_as_uint(uu),
                         mapa_u32(bar_base + 8u * (uint32_t)j, (uint32_t)lane));
        if (lane == 0) {
            z[row] = zz;
            u[row] = uu;
        }
    };

    const int nr = crank < b ? (b - crank + C - 1) / C : 0;        // rows of each block dealt to this CTA
    const int group = warp / kGroupWarps, wg = warp % kGroupWarps;
    if (nr >= kGroupWarps) {
        // a warp owns whole rows
        for (int j = group; j < s; j += kChainGroups) {
            for (int rho = wg; rho < nr; rho += kGroupWarps) {
                const int row = j * b + crank + rho * C;
                const float rr = ld_dep(r + row), yy = ld_dep(yI + row);
                const float acc = dot_chunks(row, j * b, 0, 1);
                publish(j, row, warp_sum(acc), rr, yy);
            }
        }
    } else if (nr > 0) {
        // wpr warps share a row: warp h of the row takes chunks e = h, h + wpr, ...; h = 0 (which holds the newest
        // chunk) is the lead and adds the others' partial sums
        const int wpr = kGroupWarps / nr;
        const int rho = wg / wpr, h = wg % wpr;
        if (rho < nr) {
            for (int j = group, it = 0; j < s; j += kChainGroups, ++it) {
                const int row = j * b + crank + rho * C;
                if (h == 0) {
                    const float rr = ld_dep(r + row), yy = ld_dep(yI + row);
                    float acc = dot_chunks(row, j * b, 0, wpr);
                    if (lane >= 1 && lane < wpr) {                          // lane hh collects helper hh's partial
                        while (pflag[it & 1][warp + lane] != j) { }
                        acc += part[it & 1][warp + lane];
                        cons[warp + lane] = j;
                    }
                    __syncwarp();
                    publish(j, row, warp_sum(acc), rr, yy);
                } else {
                    const float p = warp_sum(dot_chunks(row, j * b, h, wpr));
                    if (lane == 0) {
                        while (cons[warp] < j - 2 * kChainGroups) { }       // this slot's previous value has been read
                        part[it & 1][warp] = p;
                        __threadfence_block();
                        pflag[it & 1][warp] = j;
                    }
                    __syncwarp();
                }
            }
        }
    }
    __syncthreads();
    cluster_sync_all();                                 // no CTA leaves while others may still store into it
    stamp_end(stamp);
}

int recurrence_grid_ctas(const RecWorkspace &ws, int32_t sb)
{
    return std::max(1, std::min(ws.max_ctas, (sb + kRecWarps - 1) / kRecWarps));
}

template <int LOSS>
static cudaError_t launch_grid(cudaStream_t st, const float *G, int32_t ldg, const float *r, const float *yI, int32_t s,
                               int32_t b, float alpha, float *z, float *u, const RecWorkspace &ws)
{
    const int sb = s * b;
    const int grid = recurrence_grid_ctas(ws, sb);
    const int W = grid * kRecWarps;
    const int maxr = (sb + W - 1) / W;
    const bool vec = (b % 4 == 0) && (ldg % 4 == 0);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(kRecThreads);
    cfg.dynamicSmemBytes = sizeof(float) * (size_t)sb;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;        // every CTA must be resident: they wait on each other
    attr[0].val.cooperative = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    auto go = [&](auto kern) {
        return cudaLaunchKernelEx(&cfg, kern, G, ldg, r, yI, s, b, alpha, z, u, ws.utag, ws.nrep, ws.epoch, ws.done, g_stamp);
    };
    if (maxr <= 2) return vec ? go(recurrence_grid_kernel<LOSS, 2, true>) : go(recurrence_grid_kernel<LOSS, 2, false>);
    if (maxr <= 4) return vec ? go(recurrence_grid_kernel<LOSS, 4, true>) : go(recurrence_grid_kernel<LOSS, 4, false>);
    if (maxr <= 8) return vec ? go(recurrence_grid_kernel<LOSS, 8, true>) : go(recurrence_grid_kernel<LOSS, 8, false>);
    return vec ? go(recurrence_grid_kernel<LOSS, 16, true>) : go(recurrence_grid_kernel<LOSS, 16, false>);
}

template <int LOSS>
static cudaError_t launch_cluster(cudaStream_t st, const float *G, int32_t ldg, const float *r, const float *yI,
                                  int32_t s, int32_t b, float alpha, float *z, float *u, int cluster)
{
    return launch_pdl(recurrence_cluster_kernel<LOSS>, dim3(cluster), dim3(kChainThreads),
                      sizeof(float) * (size_t)s * b + 8 * (size_t)s, st, cluster, G, ldg, r, yI, s, b, alpha, z, u, g_stamp);
}

template <int LOSS>
static int cluster_size_for()
{
    auto kern = recurrence_cluster_kernel<LOSS>;
    const int smem = CASGD_MAX_SB * (int)sizeof(float) + 8 * (CASGD_MAX_SB / 4);   // u_s + one mbarrier per block
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return 0;
    cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    for (int c : {16, 8}) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(c);
        cfg.blockDim = dim3(kChainThreads);
        cfg.dynamicSmemBytes = smem;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = c;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        int n = 0;
        if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) == cudaSuccess && n >= 1) return c;
    }
    cudaGetLastError();
    return 0;
}

// Largest cluster (16, else 8, else 0) the three instantiations of the cluster kernel can run with.
int recurrence_cluster_size()
{
    const int a = cluster_size_for<CASGD_LOGISTIC>(), b = cluster_size_for<CASGD_LINEAR>(),
              c = cluster_size_for<CASGD_POISSON>();
    return std::min(a, std::min(b, c));
}

int recurrence_max_coresident_ctas(int num_sms)
{
    int per_sm = 0;
    if (cudaFuncSetAttribute(recurrence_grid_kernel<CASGD_LOGISTIC, 16, true>,
                             cudaFuncAttributeMaxDynamicSharedMemorySize, CASGD_MAX_SB * (int)sizeof(float)) != cudaSuccess)
        return 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, recurrence_grid_kernel<CASGD_LOGISTIC, 16, true>,
                                                      kRecThreads, CASGD_MAX_SB * sizeof(float)) != cudaSuccess || per_sm < 1)
        return 0;
    return num_sms;                                     // one CTA per SM
}

template <int LOSS>
static cudaError_t configure_loss()
{
    const int cap = CASGD_MAX_SB * (int)sizeof(float);
    cudaError_t e = cudaFuncSetAttribute(recurrence_cta_kernel<LOSS>, cudaFuncAttributeMaxDynamicSharedMemorySize, cap);
    auto set = [&](auto kern) {
        if (e == cudaSuccess) e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, cap);
    };
    set(recurrence_grid_kernel<LOSS, 2, true>);  set(recurrence_grid_kernel<LOSS, 2, false>);
    set(recurrence_grid_kernel<LOSS, 4, true>);  set(recurrence_grid_kernel<LOSS, 4, false>);
    set(recurrence_grid_kernel<LOSS, 8, true>);  set(recurrence_grid_kernel<LOSS, 8, false>);
    set(recurrence_grid_kernel<LOSS, 16, true>); set(recurrence_grid_kernel<LOSS, 16, false>);
    return e;
}

// (the cluster kernel's attributes are set by recurrence_cluster_size(), which casgd_init calls on every device)
cudaError_t recurrence_configure()
{
    cudaError_t e = configure_loss<CASGD_LOGISTIC>();
    if (e == cudaSuccess) e = configure_loss<CASGD_LINEAR>();
    if (e == cudaSuccess) e = configure_loss<CASGD_POISSON>();
    return e;
}

// the chain-CTA kernel (5): asked for, or ... (see recurrence_kernel_choice)
static bool chain_preferred(int32_t s, int32_t b, int32_t ldg, const RecWorkspace &ws, int impl)
{
    return impl == 5 && recurrence_chain_ok(s, b, ldg, ws.cluster);
}

bool recurrence_fuses_update(int32_t s, int32_t b, int32_t ldg, int32_t ldy, const RecWorkspace &ws, int impl)
{
    // with the update fused in, the cluster kernel beats the one-CTA kernel + a gradient kernel even for tiny G (measured)
    if (chain_preferred(s, b, ldg, ws, impl)) return recurrence_chain_fuses_update(s, b, ldy);
    return (impl >= 4 || impl == 0) && recurrence_stream_ok(s, b, ldg, ws.cluster) && recurrence_stream_fuses_update(s, b, ldy, ws.cluster);
}

// Which kernel launch_recurrence runs for this shape: 1 = one CTA, 2 = all SMs (cooperative), 3 = one cluster with
// plain loads, 4 = the streaming cluster kernel, 5 = the chain-CTA cluster kernel (small blocks).
int recurrence_kernel_choice(int32_t s, int32_t b, int32_t ldg, const RecWorkspace &ws, int impl, bool fused)
{
    const int64_t gl_bytes = 2ll * b * b * s * (s - 1);
    const int sb = s * b;
    // MAXR = 16 rows per warp covers CASGD_MAX_SB on >= 128 SMs; on fewer co-resident CTAs fall back
    const bool grid_ok = ws.max_ctas > 0 && (int64_t)ws.max_ctas * kRecWarps * 16 >= sb;
    const bool cluster_ok = ws.cluster > 0 && b % 4 == 0 && ldg % 4 == 0;
    if (chain_preferred(s, b, ldg, ws, impl)) return 5;
    const bool stream_ok = (impl >= 4 || impl == 0) && recurrence_stream_ok(s, b, ldg, ws.cluster);
    if (stream_ok && (impl >= 4 || gl_bytes >= ws.grid_threshold_bytes || fused)) return 4;
    if (cluster_ok && (impl >= 3 || (impl == 0 && gl_bytes >= ws.grid_threshold_bytes))) return 3;
    if (grid_ok && (impl >= 2 || (impl == 0 && gl_bytes >= ws.grid_threshold_bytes))) return 2;
    return 1;
}

int launch_recurrence(cudaStream_t st, const float *G, int32_t ldg, const float *r, const float *yI, int32_t s,
                      int32_t b, float alpha, int loss, float *z, float *u, const RecWorkspace &ws, int impl,
                      const FusedUpdate *fu)
{
    const int choice = recurrence_kernel_choice(s, b, ldg, ws, impl, fu != nullptr);
    if (choice == 5) return launch_recurrence_chain(st, G, ldg, r, yI, s, b, alpha, loss, z, u, fu, ws.late_trigger);
    if (choice == 4)
        return launch_recurrence_stream(st, G, ldg, r, yI, s, b, alpha, loss, z, u, ws.cluster, fu,
                                        (ws.late_trigger ? 1 : 0) | (ws.g_protected ? 2 : 0));
    if (choice == 3) {
        cudaError_t e = loss == CASGD_LOGISTIC ? launch_cluster<CASGD_LOGISTIC>(st, G, ldg, r, yI, s, b, alpha, z, u, ws.cluster)
                      : loss == CASGD_LINEAR  ? launch_cluster<CASGD_LINEAR>(st, G, ldg, r, yI, s, b, alpha, z, u, ws.cluster)
                                              : launch_cluster<CASGD_POISSON>(st, G, ldg, r, yI, s, b, alpha, z, u, ws.cluster);
        return e == cudaSuccess ? 1 : -1;
    }
    if (choice == 2) {
        cudaError_t e = loss == CASGD_LOGISTIC ? launch_grid<CASGD_LOGISTIC>(st, G, ldg, r, yI, s, b, alpha, z, u, ws)
                      : loss == CASGD_LINEAR  ? launch_grid<CASGD_LINEAR>(st, G, ldg, r, yI, s, b, alpha, z, u, ws)
                                              : launch_grid<CASGD_POISSON>(st, G, ldg, r, yI, s, b, alpha, z, u, ws);
        return e == cudaSuccess ? 1 : -1;
    }
    const size_t smem = sizeof(float) * (size_t)s * b;
    const int threads = (b >= 32) ? 1024 : 32 * ((b < 4) ? 4 : b);
    auto go = [&](auto kern) {
        return launch_pdl(kern, dim3(1), dim3(threads), smem, st, 1, G, ldg, r, yI, s, b, alpha, z, u, g_stamp);
    };
    const cudaError_t e = loss == CASGD_LOGISTIC ? go(recurrence_cta_kernel<CASGD_LOGISTIC>)
                        : loss == CASGD_LINEAR  ? go(recurrence_cta_kernel<CASGD_LINEAR>)
                                                : go(recurrence_cta_kernel<CASGD_POISSON>);
    return e == cudaSuccess ? 1 : -1;
}

}  // namespace casgd

// partition.cu -- the pieces of Alg. 1 line 5 for P > 1 ranks in the paper's 1-D block-column
// partition (L33, L141): every rank holds a column slab A[:, c0:c1] and the matching slab of x, forms its local
// r_loc = Y_loc x_loc and G_loc = Y_loc Y_loc^T, and ONE sum over the ranks of [r; G] -- sb + (sb)^2 words in Table 2
// (L154), of which only the strict block-lower part of G is ever read (L180) -- gives every rank the full r and G;
// the recurrence then runs redundantly on every rank and each rank updates its own slab of x.
//
// Payload of one outer iteration (what is summed), FP32, contiguous:
//   [ r_0 .. r_{sb-1} | block row 1 of G (b x b) | block row 2 (b x 2b) | ... | block row s-1 (b x (s-1)b) ]
// i.e. entry (i, k) of G with block(k) < block(i) = j sits at  sb + b^2 j (j-1) / 2 + (i - j b) * j b + k.
// Count = sb + b^2 s (s-1) / 2: half of Table 2's (sb)^2, because G is symmetric and only k < j blocks are used.
#include "common.cuh"

namespace casgd {

namespace {

// one warp per row of G: row i of block j >= 1 owns j*b payload words
template <bool PACK>
__global__ void __launch_bounds__(256)
payload_kernel(float *G, int32_t ldg, float *r, int32_t s, int32_t b, float *payload)
{
    pdl_trigger();
    pdl_wait();
    const int sb = s * b;
    const int gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31, W = (gridDim.x * blockDim.x) >> 5;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < sb; i += gridDim.x * blockDim.x) {
        if (PACK) payload[i] = r[i];
        else r[i] = payload[i];
    }
    for (int i = b + gw; i < sb; i += W) {
        const int j = i / b, len = j * b;
        float *row = G + (int64_t)i * ldg;
        float *dst = payload + sb + (int64_t)b * b * j * (j - 1) / 2 + (int64_t)(i - j * b) * len;
        for (int k = lane; k < len; k += 32) {
            if (PACK) dst[k] = row[k];
            else row[k] = dst[k];
        }
    }
}

constexpr int kMaxPeers = 64;
struct PeerList {
    const float *p[kMaxPeers];
};

// out[i] = sum over ranks, in rank order (every rank computes the same bits, so the redundant recurrences agree).
// The peers' buffers may be peer-mapped device memory of other GPUs (NVLink loads): a one-shot all-reduce in which
// each rank reads every peer's payload once.
__global__ void __launch_bounds__(256)
reduce_peers_kernel(const PeerList peers, int32_t P, float *out, int64_t count)
{
    pdl_trigger();
    pdl_wait();
    const int64_t nvec = count >> 2;
    for (int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; v < nvec; v += (int64_t)gridDim.x * blockDim.x) {
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int q = 0; q < P; ++q) {
            const float4 t = *reinterpret_cast<const float4 *>(peers.p[q] + 4 * v);
            acc.x += t.x; acc.y += t.y; acc.z += t.z; acc.w += t.w;
        }
        *reinterpret_cast<float4 *>(out + 4 * v) = acc;
    }
    for (int64_t i = 4 * nvec + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (int64_t)gridDim.x * blockDim.x) {
        float acc = 0.f;
        for (int q = 0; q < P; ++q) acc += peers.p[q][i];
        out[i] = acc;
    }
}

// The same sum written straight into the recurrence's inputs (G rows with stride ldg, r): reduce and unpack in one
// pass -- every rank reads each peer's payload once over NVLink and nothing is staged.
__global__ void __launch_bounds__(256)
reduce_unpack_kernel(const PeerList peers, int32_t P, float *G, int32_t ldg, float *r, int32_t s, int32_t b)
{
    pdl_trigger();
    pdl_wait();
    const int sb = s * b;
    const int gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31, W = (gridDim.x * blockDim.x) >> 5;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < sb; i += gridDim.x * blockDim.x) {
        float acc = 0.f;
        for (int q = 0; q < P; ++q) acc += peers.p[q][i];
        r[i] = acc;
    }
    for (int i = b + gw; i < sb; i += W) {
        const int j = i / b, len = j * b;
        const int64_t off = sb + (int64_t)b * b * j * (j - 1) / 2 + (int64_t)(i - j * b) * len;
        float *row = G + (int64_t)i * ldg;
        for (int k = lane; k < len; k += 32) {
            float acc = 0.f;
            for (int q = 0; q < P; ++q) acc += peers.p[q][off + k];
            row[k] = acc;
        }
    }
}

}  // namespace

int64_t payload_count(int32_t s, int32_t b) { return (int64_t)s * b + (int64_t)b * b * s * (s - 1) / 2; }

int launch_payload_pack(cudaStream_t st, const float *G, int32_t ldg, const float *r, int32_t s, int32_t b, float *payload,
                        int num_sms)
{
    const int blocks = std::max(1, std::min(4 * num_sms, (s * b * 32 + 255) / 256));
    launch_pdl(payload_kernel<true>, dim3(blocks), dim3(256), 0, st, 1, const_cast<float *>(G), ldg, const_cast<float *>(r), s, b,
               payload);
    return 1;
}

int launch_payload_unpack(cudaStream_t st, float *G, int32_t ldg, float *r, int32_t s, int32_t b, const float *payload,
                          int num_sms)
{
    const int blocks = std::max(1, std::min(4 * num_sms, (s * b * 32 + 255) / 256));
    launch_pdl(payload_kernel<false>, dim3(blocks), dim3(256), 0, st, 1, G, ldg, r, s, b, const_cast<float *>(payload));
    return 1;
}

// Returns kernels launched, or -1 when P is out of range / a buffer is misaligned.
int launch_reduce_peers(cudaStream_t st, const float *const *peers_host, int32_t P, float *out, int64_t count, int num_sms)
{
    if (P < 1 || P > kMaxPeers || ((uintptr_t)out & 15)) return -1;
    PeerList pl{};
    for (int q = 0; q < P; ++q) {
        if (!peers_host[q] || ((uintptr_t)peers_host[q] & 15)) return -1;
        pl.p[q] = peers_host[q];
    }
    const int blocks = (int)std::max<int64_t>(1, std::min<int64_t>(8 * num_sms, (count / 4 + 255) / 256));
    launch_pdl(reduce_peers_kernel, dim3(blocks), dim3(256), 0, st, 1, pl, P, out, count);
    return 1;
}

// Sum the peers' payloads straight into G and r. Returns kernels launched, or -1.
int launch_reduce_unpack(cudaStream_t st, const float *const *peers_host, int32_t P, float *G, int32_t ldg, float *r, int32_t s,
                         int32_t b, int num_sms)
{
    if (P < 1 || P > kMaxPeers) return -1;
    PeerList pl{};
    for (int q = 0; q < P; ++q) {
        if (!peers_host[q]) return -1;
        pl.p[q] = peers_host[q];
    }
    const int blocks = std::max(1, std::min(8 * num_sms, (s * b * 32 + 255) / 256));
    launch_pdl(reduce_unpack_kernel, dim3(blocks), dim3(256), 0, st, 1, pl, P, G, ldg, r, s, b);
    return 1;
}

}  // namespace casgd

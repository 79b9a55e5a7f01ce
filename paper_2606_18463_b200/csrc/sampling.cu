// sampling.cu -- Alg. 1 line 1: the s*b row indices of an outer step, drawn on the device
// i.i.d. uniformly WITH replacement. Counter-based, so a step's indices depend only on (seed, step number, position):
//   index t of outer step h:  counter = (t / 4, h mod 2^32, h div 2^32, 0xCA5D), key = (seed mod 2^32, seed div 2^32),
//   w = Philox4x32-10(counter, key)[t mod 4],  idx = floor(w * m / 2^32)
// (Philox4x32-10: Salmon et al., "Parallel random numbers: as easy as 1, 2, 3", SC'11; the multiply-shift map has a
// bias below m / 2^32). The oracle implements the same definition independently; parity is bit-exact.
#include "common.cuh"

namespace casgd {

namespace {

__device__ __forceinline__ void philox_round(uint32_t (&c)[4], uint32_t k0, uint32_t k1)
{
    const uint32_t hi0 = __umulhi(0xD2511F53u, c[0]), lo0 = 0xD2511F53u * c[0];
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c[2]), lo1 = 0xCD9E8D57u * c[2];
    const uint32_t n0 = hi1 ^ c[1] ^ k0, n2 = hi0 ^ c[3] ^ k1;
    c[0] = n0; c[1] = lo1; c[2] = n2; c[3] = lo0;
}

// one thread per group of four consecutive indices of one step
__global__ void __launch_bounds__(256)
sample_indices_kernel(int32_t *idx, int64_t n_steps, int32_t sb, int64_t m, uint64_t seed, uint64_t first_step)
{
    pdl_trigger();
    pdl_wait();                                     // the index buffer may still be read by the previous call's steps
    const int32_t groups = (sb + 3) >> 2;
    const int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= n_steps * groups) return;
    const int64_t hs = g / groups;
    const uint32_t q = (uint32_t)(g - hs * groups);
    const uint64_t h = first_step + (uint64_t)hs;
    uint32_t c[4] = {q, (uint32_t)h, (uint32_t)(h >> 32), 0xCA5Du};
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        philox_round(c, k0, k1);
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    int32_t *out = idx + hs * sb + 4 * (int64_t)q;
#pragma unroll
    for (int e = 0; e < 4; ++e)
        if (4 * (int32_t)q + e < sb) out[e] = (int32_t)(((uint64_t)c[e] * (uint64_t)m) >> 32);
}

}  // namespace

int launch_sample_indices(cudaStream_t st, int32_t *idx, int64_t n_steps, int32_t sb, int64_t m, uint64_t seed,
                          uint64_t first_step)
{
    const int64_t total = n_steps * ((sb + 3) >> 2);
    launch_pdl(sample_indices_kernel, dim3((unsigned)((total + 255) / 256)), dim3(256), 0, st, 1, idx, n_steps, sb, m, seed,
               first_step);
    return 1;
}

}  // namespace casgd

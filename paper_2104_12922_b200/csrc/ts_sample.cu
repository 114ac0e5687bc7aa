// ts_sample.cu -- S1: counter-based Philox parameter sampler, and the S12 noise-word debug export.
// P:L94 (deterministic RNG, noise included), P:L143 (uniform in the normalised range); D3, D4, D5.
#include "ts_common.cuh"

// One thread per (voice, Philox block).  Blocks 0..19 carry the 78 parameters (stream 0, words 78
// and 79 unused), block 20 is the noise-key block (stream 2).  320-byte records: thread i of a voice
// writes the 16 bytes at offset 16*i, so a warp writes 512 contiguous bytes.
__global__ void __launch_bounds__(256) ts_sample_kernel(uint64_t seed, uint64_t g0, int B, ts_voice *params) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (int64_t)B * 20) return;
    const int b = (int)(t / 20), i = (int)(t % 20);
    const uint64_t g = g0 + (uint64_t)b;
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    uint32_t w[4];
    ts_philox4x32_10((uint32_t)i, (uint32_t)g, (uint32_t)(g >> 32), 0u, k0, k1, w);
    float4 v;
    v.x = (float)(w[0] >> 8) * (1.0f / 16777216.0f);
    v.y = (float)(w[1] >> 8) * (1.0f / 16777216.0f);
    v.z = (float)(w[2] >> 8) * (1.0f / 16777216.0f);
    v.w = (float)(w[3] >> 8) * (1.0f / 16777216.0f);
    float4 *rec = reinterpret_cast<float4 *>(params + b);
    if (i == 19) {
        // words 76, 77 are parameters; the last 8 bytes of the record are noise_key (D4)
        uint32_t nk[4];
        ts_philox4x32_10(0u, (uint32_t)g, (uint32_t)(g >> 32), 2u, k0, k1, nk);
        v.z = __uint_as_float(nk[0]);
        v.w = __uint_as_float(nk[1]);
    }
    rec[i] = v;
}

cudaError_t ts_launch_sample(uint64_t seed, uint64_t g0, int B, ts_voice *d_params, cudaStream_t st) {
    const int64_t n = (int64_t)B * 20;
    const int threads = 256;
    const unsigned blocks = (unsigned)((n + threads - 1) / threads);
    ts_sample_kernel<<<blocks, threads, 0, st>>>(seed, g0, B, d_params);
    return cudaGetLastError();
}

// S12: word (n & 3) of Philox(key, ctr = (n >> 2, 0, 0, 1)).
__global__ void ts_noise_debug_kernel(uint32_t k0, uint32_t k1, uint64_t n0, int count, uint32_t *out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    const uint64_t n = n0 + (uint64_t)i;
    uint32_t w[4];
    ts_philox4x32_10((uint32_t)(n >> 2), 0u, 0u, 1u, k0, k1, w);
    out[i] = w[n & 3];
}

cudaError_t ts_launch_noise_debug(uint32_t k0, uint32_t k1, uint64_t n0, int count, uint32_t *d_out, cudaStream_t st) {
    ts_noise_debug_kernel<<<(count + 255) / 256, 256, 0, st>>>(k0, k1, n0, count, d_out);
    return cudaGetLastError();
}

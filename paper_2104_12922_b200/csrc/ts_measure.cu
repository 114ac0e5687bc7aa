// ts_measure.cu -- measurement aids (not on the hot path): a store-only fill kernel, and the issue rate of the
// instruction kinds the audio kernel is made of.  The guides give nominal lane counts; the rates that decide the audio
// kernel's ALU bound (IMAD.WIDE of the Philox rounds, packed FFMA2, MUFU, fp64) are measured here on the GPU the
// bench runs on, so that DESIGN.md's bound is derived from measurements and `bench.py` can print them beside it.
#include "ts_common.cuh"

namespace {

// store-only fill: what a pure 128-bit store stream reaches on this GPU, beside the copy peak
__global__ void __launch_bounds__(256) ts_fill_kernel(float4 *__restrict__ dst, size_t n16) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += stride) dst[i] = make_float4(0.f, 0.f, 0.f, 0.f);
}

constexpr int PIPE_ITERS = 128;   // loop iterations
constexpr int PIPE_UNROLL = 8;    // repetitions of the 8-chain group per iteration: 64 instructions against ~3 of loop overhead
typedef unsigned long long u64;

// 8 independent dependency chains per thread, 8 warps per SM sub-partition: throughput, not latency
template <int OP>
__global__ void __launch_bounds__(1024, 1) ts_pipe_kernel(u64 *__restrict__ sink, float cf, double cd, uint32_t cu, long long *__restrict__ cycles) {
    u64 a[8];
    float f[8];
    double d[8];
    uint32_t u[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        a[i] = 0x3f8000003f800000ull + i + threadIdx.x;
        f[i] = cf + i;
        d[i] = cd + i;
        u[i] = cu + i * 77 + threadIdx.x;
    }
    __syncthreads();
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < PIPE_ITERS; ++it) {
#pragma unroll
        for (int r = 0; r < PIPE_UNROLL; ++r) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (OP == 0) asm volatile("fma.rn.f32 %0, %0, %1, %1;" : "+f"(f[i]) : "f"(cf));
                if (OP == 1) asm volatile("fma.rn.f32x2 %0, %0, %1, %1;" : "+l"(a[i]) : "l"(0x3f8000003f800000ull));
                if (OP == 2) asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(a[i]) : "r"((uint32_t)a[i]), "r"(cu));
                if (OP == 3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(u[i]) : "r"(cu), "r"(u[(i + 1) & 7]));
                if (OP == 4) asm volatile("fma.rn.f64 %0, %0, %1, %1;" : "+d"(d[i]) : "d"(cd));
                if (OP == 5) asm volatile("sin.approx.ftz.f32 %0, %0;" : "+f"(f[i]));
                if (OP == 6) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(f[i]));
                if (OP == 7) asm volatile("cvt.rn.f32.s32 %0, %1;" : "=f"(f[i]) : "r"(__float_as_int(f[i])));
            }
        }
    }
    const long long t1 = clock64();
    u64 s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += a[i] + __float_as_uint(f[i]) + (u64)d[i] + u[i];
    if (s == 0x123456789ull) sink[threadIdx.x] = s;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

template <int OP> cudaError_t run_pipe(u64 *sink, long long *cycles, cudaStream_t st) {
    ts_pipe_kernel<OP><<<8, 1024, 0, st>>>(sink, 1.0001f, 1.0000001, 0x9E3779B9u, cycles);
    ts_pipe_kernel<OP><<<8, 1024, 0, st>>>(sink, 1.0001f, 1.0000001, 0x9E3779B9u, cycles);
    return cudaGetLastError();
}

}  // namespace

cudaError_t ts_launch_fill(void *d_dst, size_t bytes, cudaStream_t st) {
    ts_fill_kernel<<<148 * 32, 256, 0, st>>>(static_cast<float4 *>(d_dst), bytes / 16);
    return cudaGetLastError();
}

// host_rates[k] = cycles per warp instruction per SM sub-partition with 8 warps per sub-partition issuing only that kind:
// 0 FFMA, 1 FFMA2, 2 IMAD.WIDE.U32, 3 LOP3, 4 DFMA, 5 MUFU.SIN (with its range-reduction FMUL), 6 MUFU.EX2, 7 I2FP
cudaError_t ts_measure_pipes(double host_rates[TS_NPIPES], cudaStream_t st) {
    u64 *sink = nullptr;
    long long *cycles = nullptr;
    cudaError_t e = cudaMalloc(&sink, 1024 * sizeof(u64));
    if (e != cudaSuccess) return e;
    e = cudaMalloc(&cycles, 8 * sizeof(long long));
    if (e != cudaSuccess) { cudaFree(sink); return e; }
    for (int op = 0; op < TS_NPIPES && e == cudaSuccess; ++op) {
        switch (op) {
            case 0: e = run_pipe<0>(sink, cycles, st); break;
            case 1: e = run_pipe<1>(sink, cycles, st); break;
            case 2: e = run_pipe<2>(sink, cycles, st); break;
            case 3: e = run_pipe<3>(sink, cycles, st); break;
            case 4: e = run_pipe<4>(sink, cycles, st); break;
            case 5: e = run_pipe<5>(sink, cycles, st); break;
            case 6: e = run_pipe<6>(sink, cycles, st); break;
            default: e = run_pipe<7>(sink, cycles, st); break;
        }
        if (e != cudaSuccess) break;
        long long h[8];
        e = cudaMemcpyAsync(h, cycles, sizeof h, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        double avg = 0;
        for (int i = 0; i < 8; ++i) avg += (double)h[i] / 8.0;
        const double winst = (double)PIPE_ITERS * PIPE_UNROLL * 8 * (1024 / 32) / 4;  // warp instructions per sub-partition
        host_rates[op] = avg / winst;
    }
    cudaFree(sink);
    cudaFree(cycles);
    return e;
}

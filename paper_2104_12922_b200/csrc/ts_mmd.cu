// ts_mmd.cu -- maximum mean discrepancy with the l1 core distance (Eq. 2 at P:L230; reading D25):
//     MMD(X, Y) = (1/n^2) sum_{i,j} [ 2 |x_i - y_j|_1 - |x_i - x_j|_1 - |y_i - y_j|_1 ]
// over two sets of n embeddings of dimension d (the paper: n = 1000 sounds, d = 512 OpenL3 values).
// An l1 distance is not a contraction (no product to accumulate), so there is nothing here for the tensor cores:
// the work is 2 FADD-class instructions per (pair, component) -- a subtraction and an accumulation of its absolute
// value -- on the fp32 pipes.  Bound: 2 n_pairs d thread instructions against 148 SMs x 128 lanes per clock; the 4 MB
// of embeddings stay in L2 and are re-used from shared memory (64 x 64 pairs per CTA, 4 x 4 per thread).
// The three pair matrices are tiled in one grid; X-X and Y-Y are symmetric, so only tiles on or above the diagonal
// are computed and the off-diagonal ones count twice.  Per-pair sums are fp32, sums over pairs fp64 in a fixed order
// (per-CTA partials, then one CTA adds them): bitwise reproducible.
#include "ts_common.cuh"

namespace {

constexpr int MT = 64;   // pairs per tile side
constexpr int MK = 32;   // components per shared-memory chunk
constexpr int MTHREADS = 256;
constexpr int MSPLIT = 4;  // CTAs per tile, each over a quarter of the components: 2112 CTAs at n = 1000 (4.8 waves)

// tile list: [0, T*T) X-Y tiles (ti, tj); then T(T+1)/2 X-X tiles with tj >= ti; then as many Y-Y tiles
__device__ __forceinline__ void ts_mmd_tile(int t, int T, int &m, int &ti, int &tj) {
    const int tri = T * (T + 1) / 2;
    if (t < T * T) { m = 0; ti = t / T; tj = t - ti * T; return; }
    t -= T * T;
    m = 1;
    if (t >= tri) { t -= tri; m = 2; }
    int r = 0;  // row r holds T - r tiles
    while (t >= T - r) { t -= T - r; ++r; }
    ti = r;
    tj = r + t;
}

__global__ void __launch_bounds__(MTHREADS)
ts_mmd_tiles_kernel(const float *__restrict__ X, const float *__restrict__ Y, int n, int d, int T, double *__restrict__ partial) {
    // component-major: a thread's four rows are one 128-bit load; rows padded by 4 floats so that the transposing stores
    // (32 lanes = 32 components of one row) spread over 8 banks instead of hitting one
    __shared__ __align__(16) float As[MK][MT + 4];
    __shared__ __align__(16) float Bs[MK][MT + 4];
    __shared__ double red[MTHREADS / 32];
    int m, ti, tj;
    ts_mmd_tile((int)blockIdx.x, T, m, ti, tj);
    const float *A = (m == 2) ? Y : X;
    const float *Bm = (m == 1) ? X : Y;
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    const int i0 = ti * MT, j0 = tj * MT;
    float acc[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b] = 0.f;

    // this CTA's share of the components: chunks of MK, dealt round-robin over the MSPLIT CTAs of the tile
    for (int k0 = (int)blockIdx.y * MK; k0 < d; k0 += MK * MSPLIT) {
        // 64 rows x 32 components of each operand; a thread loads component (tid % 32) of rows tid / 32 + 8 p
#pragma unroll
        for (int p = 0; p < MT / 8; ++p) {
            const int r = (tid >> 5) + 8 * p, k = k0 + (tid & 31);
            As[tid & 31][r] = (i0 + r < n && k < d) ? __ldg(A + (size_t)(i0 + r) * d + k) : 0.f;
            Bs[tid & 31][r] = (j0 + r < n && k < d) ? __ldg(Bm + (size_t)(j0 + r) * d + k) : 0.f;
        }
        __syncthreads();
#pragma unroll 8
        for (int kk = 0; kk < MK; ++kk) {
            const float4 a = *reinterpret_cast<const float4 *>(&As[kk][ty * 4]);
            const float4 b = *reinterpret_cast<const float4 *>(&Bs[kk][tx * 4]);
            const float av[4] = {a.x, a.y, a.z, a.w}, bv[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
            for (int p = 0; p < 4; ++p)
#pragma unroll
                for (int q = 0; q < 4; ++q) acc[p][q] += fabsf(av[p] - bv[q]);
        }
        __syncthreads();
    }
    double s = 0.0;
#pragma unroll
    for (int p = 0; p < 4; ++p)
#pragma unroll
        for (int q = 0; q < 4; ++q)
            if (i0 + ty * 4 + p < n && j0 + tx * 4 + q < n) s += (double)acc[p][q];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if ((tid & 31) == 0) red[tid >> 5] = s;
    __syncthreads();
    if (tid == 0) {
        double t = 0.0;
        for (int w = 0; w < MTHREADS / 32; ++w) t += red[w];
        partial[(size_t)blockIdx.x * MSPLIT + blockIdx.y] = (m != 0 && tj > ti) ? 2.0 * t : t;  // the mirrored tile of a symmetric matrix
    }
}

// Fixed-order reduction of the per-CTA partials: thread t adds partials t, t + 256, ... of a matrix in that order, then
// the 256 thread sums are added in index order by a fixed tree -- the same bits on every run.
__global__ void __launch_bounds__(256) ts_mmd_final_kernel(const double *__restrict__ partial, int n, int T, double *__restrict__ out) {
    __shared__ double red[3][256];
    const int tri = T * (T + 1) / 2, tid = threadIdx.x;
    const int first[3] = {0, T * T * MSPLIT, (T * T + tri) * MSPLIT}, count[3] = {T * T * MSPLIT, tri * MSPLIT, tri * MSPLIT};
#pragma unroll
    for (int m = 0; m < 3; ++m) {
        double s = 0.0;
        for (int i = tid; i < count[m]; i += 256) s += partial[first[m] + i];
        red[m][tid] = s;
    }
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (tid < o)
#pragma unroll
            for (int m = 0; m < 3; ++m) red[m][tid] += red[m][tid + o];
        __syncthreads();
    }
    if (tid == 0) {
        const double sxy = red[0][0], sxx = red[1][0], syy = red[2][0];
        out[0] = (2.0 * sxy - sxx - syy) / ((double)n * (double)n);
        out[1] = sxy;
        out[2] = sxx;
        out[3] = syy;
    }
}

}  // namespace

size_t ts_mmd_partial_count(int n) {
    const size_t T = ((size_t)n + MT - 1) / MT;
    return (T * T + T * (T + 1)) * MSPLIT;
}

cudaError_t ts_launch_mmd(const float *d_x, const float *d_y, int n, int d, double *d_partial, double *d_out, cudaStream_t st) {
    const int T = (n + MT - 1) / MT;
    const unsigned tiles = (unsigned)(T * T + T * (T + 1));
    ts_mmd_tiles_kernel<<<dim3(tiles, MSPLIT), MTHREADS, 0, st>>>(d_x, d_y, n, d, T, d_partial);
    ts_mmd_final_kernel<<<1, 256, 0, st>>>(d_partial, n, T, d_out);
    return cudaGetLastError();
}

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

// ---- the sorted form: O(d n log^2 n) instead of O(d n^2) -----------------------------------------------------------------
// Eq. 2 needs only the SUMS of the three pair matrices, and an l1 distance is a sum over components, so
//     sum_{i,j} |x_i - y_j|_1 = sum_k sum_{i,j} |x_ik - y_jk|,
// and a one-dimensional sum of absolute differences follows from ONE sort: in ascending order every element v adds
// v * (number of smaller elements of the other set) - (their sum).  One CTA per component: the 2n values of the component
// are put on a fixed-point grid (2^-61 of the component's largest magnitude: an fp32 value is ON the grid unless it is
// more than 2^37 times smaller than that maximum), sorted by a bitonic network in shared memory with their set tag in the
// low key bit, and the counts and sums of the smaller elements come from one block scan.  Everything after the grid is
// INTEGER arithmetic (64-bit values, 128-bit sums and products): exact and associative, so the result does not depend on any summation order, MMD(X, X) is exactly 0 and the three sums
// of X = Y are equal bit for bit.  n = 1000, d = 512: 1.0e6 sorted keys instead of 1.5e9 (pair, component) items.
constexpr int SORT_THREADS = 512;
constexpr int SORT_MAX_M = 16384;  // keys per component (next power of two >= 2n): 128 KB of shared memory

typedef __int128 ts_i128;
__device__ __forceinline__ ts_i128 ts_shfl_up128(ts_i128 v, int o) {
    const unsigned long long lo = __shfl_up_sync(0xffffffffu, (unsigned long long)v, o);
    const unsigned long long hi = __shfl_up_sync(0xffffffffu, (unsigned long long)((unsigned __int128)v >> 64), o);
    return (ts_i128)(((unsigned __int128)hi << 64) | lo);
}
__device__ __forceinline__ ts_i128 ts_shfl_xor128(ts_i128 v, int o) {
    const unsigned long long lo = __shfl_xor_sync(0xffffffffu, (unsigned long long)v, o);
    const unsigned long long hi = __shfl_xor_sync(0xffffffffu, (unsigned long long)((unsigned __int128)v >> 64), o);
    return (ts_i128)(((unsigned __int128)hi << 64) | lo);
}
__device__ __forceinline__ double ts_i128_to_double(ts_i128 x) {  // two roundings, the same for the same integer
    const bool neg = x < 0;
    const unsigned __int128 m = neg ? (unsigned __int128)(-x) : (unsigned __int128)x;
    const double r = (double)(unsigned long long)(m >> 64) * 18446744073709551616.0 + (double)(unsigned long long)m;
    return neg ? -r : r;
}

#ifndef TS_MMD_MINB
#define TS_MMD_MINB 3  // 40 registers: three CTAs per SM instead of two (81 vs 94 us at n = 1000, d = 512)
#endif
__global__ void __launch_bounds__(SORT_THREADS, TS_MMD_MINB)
ts_mmd_sort_kernel(const float *__restrict__ X, const float *__restrict__ Y, int n, int d, int M, double *__restrict__ partial) {
    extern __shared__ __align__(16) unsigned long long keys[];  // M keys: (fixed-point value + 2^62) << 1 | tag (0 = X, 1 = Y)
    __shared__ float red_f[SORT_THREADS / 32];
    __shared__ ts_i128 red_i[3][SORT_THREADS / 32];
    __shared__ int red_c[2][SORT_THREADS / 32];
    const int k = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;

    // ---- the grid: 2^(61 - E) with 2^E above the largest magnitude of the component
    float mx = 0.f;
    for (int i = tid; i < 2 * n; i += SORT_THREADS) {
        const float v = (i < n) ? __ldg(X + (size_t)i * d + k) : __ldg(Y + (size_t)(i - n) * d + k);
        mx = fmaxf(mx, fabsf(v));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if (lane == 0) red_f[wid] = mx;
    __syncthreads();
    mx = red_f[0];
#pragma unroll
    for (int w = 1; w < SORT_THREADS / 32; ++w) mx = fmaxf(mx, red_f[w]);
    int E = 0;
    if (mx > 0.f) frexpf(mx, &E);  // mx = f * 2^E, f in [0.5, 1)
    const double scale = ldexp(1.0, 61 - E), inv_scale = ldexp(1.0, E - 61);
    for (int i = tid; i < M; i += SORT_THREADS) {
        unsigned long long key = ~0ull;  // padding sorts last
        if (i < 2 * n) {
            const float v = (i < n) ? __ldg(X + (size_t)i * d + k) : __ldg(Y + (size_t)(i - n) * d + k);
            const long long q = __double2ll_rn((double)v * scale);  // |q| < 2^61
            key = ((unsigned long long)(q + (1ll << 62)) << 1) | (unsigned long long)(i >= n);
        }
        keys[i] = key;
    }
    __syncthreads();

    // ---- bitonic sort, ascending.  Two levels of the network (distances j and j / 2) per pass over shared memory: a thread
    // takes the four keys i, i + j/2, i + j, i + j + j/2 and does both levels in registers (half the passes and barriers);
    // a merge with an odd number of levels ends with one single-level pass (distance 1).
    for (int kk = 2; kk <= M; kk <<= 1) {
        int j = kk >> 1;
        for (; j >= 2; j >>= 2) {
            const int h = j >> 1, lh = 31 - __clz(h);
            for (int t = tid; t < (M >> 2); t += SORT_THREADS) {
                const int i = ((t >> lh) << (lh + 2)) | (t & (h - 1));
                const bool up = (i & kk) == 0;
                unsigned long long e0 = keys[i], e1 = keys[i + h], e2 = keys[i + j], e3 = keys[i + j + h], x;
                if ((e0 > e2) == up) { x = e0; e0 = e2; e2 = x; }
                if ((e1 > e3) == up) { x = e1; e1 = e3; e3 = x; }
                if ((e0 > e1) == up) { x = e0; e0 = e1; e1 = x; }
                if ((e2 > e3) == up) { x = e2; e2 = e3; e3 = x; }
                keys[i] = e0; keys[i + h] = e1; keys[i + j] = e2; keys[i + j + h] = e3;
            }
            __syncthreads();
        }
        if (j == 1) {
            for (int t = tid; t < (M >> 1); t += SORT_THREADS) {
                const int i = 2 * t;
                const unsigned long long a = keys[i], b = keys[i + 1];
                if ((a > b) == ((i & kk) == 0)) { keys[i] = b; keys[i + 1] = a; }
            }
            __syncthreads();
        }
    }

    // ---- counts and sums of the smaller elements of each set: thread-local runs of M / 512 keys + one block scan
    const int per = M / SORT_THREADS;  // M >= 512 (the launcher pads)
    const int p0 = tid * per;
    int cx = 0, cy = 0;
    ts_i128 sx = 0, sy = 0;
    for (int i = 0; i < per; ++i) {
        const unsigned long long key = keys[p0 + i];
        if (key == ~0ull) break;
        const long long v = (long long)(key >> 1) - (1ll << 62);
        if (key & 1ull) { ++cy; sy += v; } else { ++cx; sx += v; }
    }
    int icx = cx, icy = cy;  // inclusive scans over the threads, in thread order
    ts_i128 isx = sx, isy = sy;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int a = __shfl_up_sync(0xffffffffu, icx, o), b = __shfl_up_sync(0xffffffffu, icy, o);
        const ts_i128 c = ts_shfl_up128(isx, o), e = ts_shfl_up128(isy, o);
        if (lane >= o) { icx += a; icy += b; isx += c; isy += e; }
    }
    if (lane == 31) { red_c[0][wid] = icx; red_c[1][wid] = icy; red_i[0][wid] = isx; red_i[1][wid] = isy; }
    __syncthreads();
    int bx = icx - cx, by = icy - cy;  // exclusive prefix of this thread
    ts_i128 bsx = isx - sx, bsy = isy - sy;
    for (int w = 0; w < wid; ++w) { bx += red_c[0][w]; by += red_c[1][w]; bsx += red_i[0][w]; bsy += red_i[1][w]; }
    __syncthreads();

    // ---- every element against the smaller ones: D_xy (cross pairs once), D_xx, D_yy (unordered pairs once)
    ts_i128 dxy = 0, dxx = 0, dyy = 0;
    for (int i = 0; i < per; ++i) {
        const unsigned long long key = keys[p0 + i];
        if (key == ~0ull) break;
        const ts_i128 v = (long long)(key >> 1) - (1ll << 62);
        if (key & 1ull) {
            dxy += v * bx - bsx;
            dyy += v * by - bsy;
            ++by; bsy += v;
        } else {
            dxy += v * by - bsy;
            dxx += v * bx - bsx;
            ++bx; bsx += v;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        dxy += ts_shfl_xor128(dxy, o);
        dxx += ts_shfl_xor128(dxx, o);
        dyy += ts_shfl_xor128(dyy, o);
    }
    if (lane == 0) { red_i[0][wid] = dxy; red_i[1][wid] = dxx; red_i[2][wid] = dyy; }
    __syncthreads();
    if (tid == 0) {
        ts_i128 a = 0, b = 0, c = 0;
        for (int w = 0; w < SORT_THREADS / 32; ++w) { a += red_i[0][w]; b += red_i[1][w]; c += red_i[2][w]; }
        // ordered pairs: the cross matrix holds every (x_i, y_j) once, the symmetric ones every unordered pair twice
        partial[(size_t)k * 3 + 0] = ts_i128_to_double(a) * inv_scale;
        partial[(size_t)k * 3 + 1] = ts_i128_to_double(2 * b) * inv_scale;
        partial[(size_t)k * 3 + 2] = ts_i128_to_double(2 * c) * inv_scale;
    }
}

// Fixed-order sum over the components: thread t adds components t, t + 256, ... in that order, then a fixed tree.
__global__ void __launch_bounds__(256) ts_mmd_sort_final_kernel(const double *__restrict__ partial, int n, int d, double *__restrict__ out) {
    __shared__ double red[3][256];
    const int tid = threadIdx.x;
#pragma unroll
    for (int m = 0; m < 3; ++m) {
        double s = 0.0;
        for (int k = tid; k < d; k += 256) s += partial[(size_t)k * 3 + m];
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

static int ts_mmd_sort_M(int n) {  // keys per component in the sorted form, 0 if n is too large for shared memory
    int M = SORT_THREADS;
    while (M < 2 * n && M < SORT_MAX_M) M <<= 1;
    return (M >= 2 * n) ? M : 0;
}
// Which form is faster: the bitonic network costs M log2 M (log2 M + 1) / 2 compare-exchange slots per component, the
// pairwise form n^2 pairs; measured on a B200 (d = 512: n = 1000 80 vs 110 us, n = 4000 336 vs 1466 us, n = 256 31 vs 21 us)
// one slot of the network costs about as much as six pairs.
static bool ts_mmd_sorted_is_faster(int n, int M) {
    int L = 0;
    while ((1 << L) < M) ++L;
    return 6.0 * (double)M * (double)(L * (L + 1) / 2) < (double)n * (double)n;
}

size_t ts_mmd_partial_count(int n, int d) {
    const size_t T = ((size_t)n + MT - 1) / MT;
    const size_t tiles = (T * T + T * (T + 1)) * MSPLIT, comps = (size_t)d * 3;
    return tiles > comps ? tiles : comps;
}

cudaError_t ts_launch_mmd(const float *d_x, const float *d_y, int n, int d, double *d_partial, double *d_out, int pairwise, cudaStream_t st) {
    const int M = (pairwise == 1) ? 0 : ts_mmd_sort_M(n);
    if (M && (pairwise == 2 || ts_mmd_sorted_is_faster(n, M))) {  // the sorted form
        static bool attr = false;
        if (!attr) {
            cudaError_t e = cudaFuncSetAttribute(ts_mmd_sort_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SORT_MAX_M * 8);
            if (e != cudaSuccess) return e;
            attr = true;
        }
        ts_mmd_sort_kernel<<<(unsigned)d, SORT_THREADS, (size_t)M * 8, st>>>(d_x, d_y, n, d, M, d_partial);
        ts_mmd_sort_final_kernel<<<1, 256, 0, st>>>(d_partial, n, d, d_out);
        return cudaGetLastError();
    }
    const int T = (n + MT - 1) / MT;  // the pairwise form (n > 8192, faster at this n, or asked for)
    const unsigned tiles = (unsigned)(T * T + T * (T + 1));
    ts_mmd_tiles_kernel<<<dim3(tiles, MSPLIT), MTHREADS, 0, st>>>(d_x, d_y, n, d, T, d_partial);
    ts_mmd_final_kernel<<<1, 256, 0, st>>>(d_partial, n, T, d_out);
    return cudaGetLastError();
}

// ---- ts_mmd_l1_static (tsynth.h): the same two kernels, per-CTA partial sums kept in memory the library image carries --------
// The partial sums above are the only scratch memory the MMD kernels use.  Some hosts of this library must not (or cannot)
// ask the CUDA allocator for it at call time: a process whose device memory is entirely owned by another allocator (a
// framework's caching pool sized to the whole GPU leaves a raw cudaMalloc nothing to hand out), a latency-bound audio or
// serving loop that cannot take cudaMalloc's implicit device-wide synchronisation, a plug-in running under a host that
// forbids allocation after start-up.  For them the scratch is this file-scope array: it is part of the loaded module, so
// every GPU that loads libtsynth.so holds TS_MMD_STATIC_MAX_PARTIALS * 8 bytes (256 KB) of it from module load to exit,
// whether or not the call is ever made.
// In HOST code the name `ts_mmd_static_partial` is only a handle for the runtime (a host-side shadow object): its address
// is not a device address, and a kernel handed `&ts_mmd_static_partial[0]` from host code would fault or write somewhere
// unrelated.  The device address is looked up once per device with cudaGetSymbolAddress, with that device current.
static __device__ __align__(256) double ts_mmd_static_partial[TS_MMD_STATIC_MAX_PARTIALS];

constexpr int TS_MMD_MAX_DEVICES = 64;
static double *ts_mmd_static_ptr[TS_MMD_MAX_DEVICES];  // device address of the array on each device ordinal, NULL = not looked up yet

size_t ts_mmd_static_capacity() { return (size_t)TS_MMD_STATIC_MAX_PARTIALS; }

// The caller has checked ts_mmd_partial_count(n, d) <= ts_mmd_static_capacity().  No cudaMalloc / cudaFree here or below:
// cudaGetDevice, cudaGetSymbolAddress (first call per device), cudaFuncSetAttribute (first sorted-form launch) and the
// two kernel launches are all this path calls.  Nothing in the array has to be zero on entry -- the first kernel of a call
// writes every partial its final kernel reads -- so the previous call's contents are simply overwritten.
cudaError_t ts_launch_mmd_static(const float *d_x, const float *d_y, int n, int d, double *d_out, cudaStream_t st) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool cached = dev >= 0 && dev < TS_MMD_MAX_DEVICES;
    double *scratch = cached ? ts_mmd_static_ptr[dev] : nullptr;
    if (!scratch) {  // set-up: once per device (ordinals past the cache look it up on every call)
        e = cudaGetSymbolAddress((void **)&scratch, ts_mmd_static_partial);
        if (e != cudaSuccess) return e;
        if (!scratch) return cudaErrorInvalidSymbol;
        if (cached) ts_mmd_static_ptr[dev] = scratch;
    }
    return ts_launch_mmd(d_x, d_y, n, d, scratch, d_out, 0, st);
}

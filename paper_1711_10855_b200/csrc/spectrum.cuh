// spectrum.cuh -- the step before the correlation ("the FFT output of the observation";
// DESIGN.md reading 18): the real time series of n_t = 2N samples -> its N lowest Fourier bins (eq.(3)),
// whitened in blocks of bins so that re and im have unit variance -- the input fdas_convolve expects.
//
// The 2N real samples are read as N complex numbers z[n] = x[2n] + i x[2n+1]; Z = DFT_N(z) is computed by the
// four-step decomposition N = N1 N2 on top of the batched segment FFT (fft_batch.cuh), with three tiled
// transposes (the second one also applies the twiddles w_N^{n2 k1}); one more pass separates the two interleaved
// real transforms, X_k = E_k + w_{2N}^k O_k, and whitens.  Every pass is a stream over HBM (8 bytes in, 8 bytes
// out per point); at N = 2^22 the whole chain moves about 0.5 GB, a few per cent of the correlation's time.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fdas {

// exp(i pi scale e / n) for 0 <= e < n, n a power of two, scale = -1 or -2, as float2 (cos, sin).
// For n <= 2^24 the fraction e / n is exact in float32 (e has at most 24 bits, n is a power of two) and sincospif
// reduces its argument exactly, so the result is within 1 ulp of the true root -- what rounding a double evaluation
// would give to half an ulp -- at a small fraction of its cost (the double version was 15 us of the 25 us of the
// twiddling transpose and 20 us of the 34 us of the last pass at n = 2^22; profiles/r3_spectrum.md).
// Longer transforms keep the double evaluation: there e / n does not fit a float.
__device__ __forceinline__ float2 unit_root(long long e, long long n, float scale)
{
    float s, c;
    if (n <= (1ll << 24)) {
        sincospif(scale * ((float)e * (1.0f / (float)n)), &s, &c);
    } else {
        double sd, cd;
        sincospi((double)scale * (double)e / (double)n, &sd, &cd);
        s = (float)sd;
        c = (float)cd;
    }
    return make_float2(c, s);
}

// out[c][r] = in[r][c] (* w_N^{r c} if TWIDDLE), in: [rows][cols] complex64.  32 x 32 tiles through shared memory,
// 32 x 8 threads; rows and cols are multiples of 32.
template <bool TWIDDLE>
__global__ void __launch_bounds__(256) fdas_transpose_kernel(const float2 *__restrict__ in, float2 *__restrict__ out, int rows,
                                                             int cols, long long n_total)
{
    __shared__ float2 tile[32][33];
    const int c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
    const int tx = threadIdx.x, ty = threadIdx.y;
#pragma unroll
    for (int j = 0; j < 32; j += 8) {
        const int r = r0 + ty + j, c = c0 + tx;
        float2 v = __ldcs(in + (size_t)r * cols + c);
        if (TWIDDLE) {
            // w_N^{r c} = exp(-2 pi i (r c mod N) / N)
            const long long e = ((long long)r * c) & (n_total - 1); // N is a power of two
            const float2 w = unit_root(e, n_total, -2.0f);
            v = make_float2(v.x * w.x - v.y * w.y, v.x * w.y + v.y * w.x);
        }
        tile[ty + j][tx] = v;
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < 32; j += 8) {
        const int c = c0 + ty + j, r = r0 + tx;
        __stcs(out + (size_t)c * rows + r, tile[tx][ty + j]);
    }
}

// Z (natural order, N complex) -> bins k = 0 .. N-1 of the real series' transform, whitened per block:
//   E = (Z_k + conj Z_{N-k}) / 2,  O = -i (Z_k - conj Z_{N-k}) / 2,  X_k = E + w_{2N}^k O
//   m_b = mean over the block of |X_k|^2 (bin 0 counted as 0);  A_k = X_k sqrt(2 / m_b),  A_0 = 0
// One CTA per block of blk bins (blk <= 0: no whitening, one CTA per 4096 bins).
__global__ void __launch_bounds__(256) fdas_rfft_whiten_kernel(const float2 *__restrict__ Z, float2 *__restrict__ out, long long N,
                                                               long long blk)
{
    const bool whiten = blk > 0;
    const long long width = whiten ? blk : 4096;
    const long long b0 = (long long)blockIdx.x * width;
    const long long b1 = b0 + width < N ? b0 + width : N;
    __shared__ float red[8];
    __shared__ float s_scale;
    // bin k of the real series' transform from Z_k and Z_{N-k}
    auto bin = [&](long long k) {
        const float2 zk = __ldg(Z + k);
        const float2 zc = __ldg(Z + ((N - k) & (N - 1)));       // conj applied below
        const float er = 0.5f * (zk.x + zc.x), ei = 0.5f * (zk.y - zc.y);
        const float orr = 0.5f * (zk.y + zc.y), oi = -0.5f * (zk.x - zc.x);
        const float2 w = unit_root(k, N, -1.0f);                 // w_{2N}^k = exp(-i pi k / N)
        float2 x = make_float2(er + (orr * w.x - oi * w.y), ei + (orr * w.y + oi * w.x));
        if (whiten && k == 0) x = make_float2(0.f, 0.f);
        return x;
    };
    // Blocks of up to 16 bins per thread (blk <= 4096, the usual case) stay in registers between the two phases, so the
    // spectrum is written once; wider blocks are written unscaled and rescaled in place (each thread its own bins).
    constexpr int PER = 16;
    const bool in_regs = width <= (long long)PER * blockDim.x;
    float2 xr[PER];
    float acc = 0.f;
    if (in_regs) {
#pragma unroll
        for (int i = 0; i < PER; ++i) {
            const long long k = b0 + threadIdx.x + (long long)i * blockDim.x;
            xr[i] = make_float2(0.f, 0.f);
            if (k < b1) {
                xr[i] = bin(k);
                acc += xr[i].x * xr[i].x + xr[i].y * xr[i].y;
                if (!whiten) out[k] = xr[i];
            }
        }
    } else {
        for (long long k = b0 + threadIdx.x; k < b1; k += blockDim.x) {
            const float2 x = bin(k);
            acc += x.x * x.x + x.y * x.y;
            out[k] = x;
        }
    }
    if (!whiten) return;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        float tot = 0.f;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) tot += red[w];  // fixed order: deterministic
        const float mean = tot / (float)(b1 - b0);
        s_scale = mean > 0.f ? sqrtf(2.0f / mean) : 0.f;
    }
    __syncthreads();
    const float sc = s_scale;
    if (in_regs) {
#pragma unroll
        for (int i = 0; i < PER; ++i) {
            const long long k = b0 + threadIdx.x + (long long)i * blockDim.x;
            if (k < b1) __stcs(out + k, make_float2(xr[i].x * sc, xr[i].y * sc));
        }
    } else {
        for (long long k = b0 + threadIdx.x; k < b1; k += blockDim.x) { // each thread rescales what it wrote itself
            const float2 x = out[k];
            out[k] = make_float2(x.x * sc, x.y * sc);
        }
    }
}

} // namespace fdas

// fft_batch.cuh -- the segment FFT as a stand-alone batched transform (Table 1 P:52-60:
// "calculating 100 FFTs per kernel launch, while launching 1000 of these kernels").  One CTA transforms one
// length-L sequence at a time with the same device code the convolution kernel uses for its forward transform
// (fft_device.cuh: registers + shared-memory exchanges), natural order in and out, and walks the batch with a
// grid stride.  HBM-bound when the batch is large: 8 bytes in and 8 bytes out per point.
#pragma once
#include "fft_device.cuh"

namespace fdas {

template <class C> __host__ __device__ constexpr int fft_batch_buf_elems()
{
    return C::SMEM_ELEMS > C::L + C::L / 16 ? C::SMEM_ELEMS : C::L + C::L / 16;
}
template <class C> constexpr size_t fft_batch_smem_bytes() { return 2 * sizeof(float2) * (size_t)fft_batch_buf_elems<C>(); }

// inverse != 0: the unnormalised inverse, computed as conj(DFT(conj x)) with the same forward passes
template <class C>
__global__ void __launch_bounds__(C::NT, (512 / C::NT) > 0 ? (512 / C::NT) : 1) fdas_fft_batch_kernel(const float2 *__restrict__ in, float2 *__restrict__ out,
                                                               const float2 *__restrict__ tw, long long n_fft, int inverse)
{
    constexpr int E = C::E, NT = C::NT, RL = C::R(C::P - 1), BL = E / RL;
    static_assert((C::L / RL) % 16 == 0 && NT % 16 == 0, "padding by one element per 16 must commute with the strides");
    extern __shared__ float2 smem[];
    float2 *buf0 = smem, *buf1 = smem + fft_batch_buf_elems<C>();
    const int t = threadIdx.x;
    const float sgn = inverse ? -1.f : 1.f;
    for (long long f = blockIdx.x; f < n_fft; f += gridDim.x) {
        const float2 *x = in + (size_t)f * C::L;
        float2 *y = out + (size_t)f * C::L;
        float2 v[E];
#pragma unroll
        for (int d = 0; d < E; ++d) {
            v[d] = __ldcs(x + d * NT + t);
            v[d].y *= sgn;
        }
        fwd_pass_regs<C, 0>(v, tw, t);
        __syncthreads(); // the previous sequence's reads of the exchange buffers are done
        fwd_from<C, 0, true>(v, buf0, buf1, tw, t);
        // digit-reversed registers -> natural order through shared memory (element f at f + f/16: both index
        // maps step through f in strides of 16 within a half-warp), then coalesced stores
        float2 *nat = ((C::P - 1) & 1) ? buf1 : buf0; // the buffer the last exchange did not use
#pragma unroll
        for (int b = 0; b < BL; ++b) {
            const int k0 = nat_freq<C>(t, b, 0); // register (b, d) holds frequency k0 + d L/RL, and 16 divides L/RL
            float2 *dst = nat + k0 + (k0 >> 4);
#pragma unroll
            for (int d = 0; d < RL; ++d) dst[d * (C::L / RL) + d * (C::L / RL / 16)] = v[b * RL + d];
        }
        __syncthreads();
        const float2 *src = nat + t + (t >> 4); // NT is a multiple of 16
#pragma unroll
        for (int d = 0; d < E; ++d) {
            float2 r = src[d * NT + d * (NT / 16)];
            r.y *= sgn;
            __stcs(y + d * NT + t, r);
        }
    }
}

} // namespace fdas

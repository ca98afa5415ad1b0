// fft_device.cuh -- the segment FFT of the FDAS hot path as device code (sm_100a).
//
// eq.(3), P:35 of arXiv:1711.10855:  X_m = sum_n x_n w_N^{nm},  w_N = exp(-i 2 pi / N),  computed by
// the divide-and-conquer of P:40 ("each FFT is itself composed from smaller FFTs"), with several
// elements per thread so that a thread's sub-FFTs share their twiddles -- here E = 8 or 16
// elements per thread held in registers, radix-8/16 butterflies done entirely in registers, and
// one shared-memory exchange between passes.
//
// Decomposition: L = R0*R1*...*R_{P-1}.  A point's position is the
// mixed-radix number p = ((d0*R1 + d1)*R2 + d2)..., d0 most significant.
//   forward  = decimation in frequency: pass I transforms digit I from time to frequency, then
//              multiplies by w_{R_I*Lo_I}^{k_I * low}, Lo_I = R_{I+1}*...*R_{P-1}, low = the digits
//              below I.  Natural-order input, digit-reversed output; no reordering pass.
//   inverse  = decimation in time, the exact mirror: passes P-1 ... 0 with conjugate twiddles
//              applied BEFORE each butterfly.  Digit-reversed input, natural-order output.
// In pass I ("layout I") thread t owns, for b < E/R_I, the R_I points that differ only in digit I
// and whose other digits spell o = t + b*NT.  Because R0 = E and every R_I divides R0, the address
// of (t, b, d) is base_I(t) + b*R_I*stride(0) + d*stride(I): one register per layout plus
// immediates.  Shared-memory strides are padded (stride(P-2) = R_{P-1}+1) so that every 64-bit
// access of a half-warp falls in distinct bank pairs (checked by tests/test_host_layout.py).
#pragma once
#include <cuda_runtime.h>

#include "butterflies_gen.cuh"

namespace fdas {

template <int L_, int E_, int R0_, int R1_, int R2_, int R3_>
struct CfgT {
    static constexpr int L = L_, E = E_, NT = L_ / E_;
    static constexpr int P = (R3_ > 1) ? 4 : 3;
    __host__ __device__ static constexpr int R(int i) { return i == 0 ? R0_ : i == 1 ? R1_ : i == 2 ? R2_ : R3_; }
    __host__ __device__ static constexpr int Lo(int i) { int p = 1; for (int j = i + 1; j < P; ++j) p *= R(j); return p; }
    // padded shared-memory stride of digit j, in complex elements
    __host__ __device__ static constexpr int stride(int j)
    {
        int s = 1;
        for (int k = P - 1; k > j; --k) s = s * R(k) + (k == P - 1 ? 1 : 0);
        return s;
    }
    static constexpr int SMEM_ELEMS = stride(0) * R0_; // one exchange buffer, complex elements
    static_assert(R0_ == E_, "pass 0 must be radix E");
    static_assert(R0_ * R1_ * R2_ * R3_ == L_, "radices must multiply to L");
    static_assert(E_ % R1_ == 0 && E_ % R2_ == 0 && E_ % R3_ == 0, "radices must divide E");
};

template <int L> struct Cfg;
template <> struct Cfg<512>  : CfgT<512, 8, 8, 8, 8, 1> {};
template <> struct Cfg<1024> : CfgT<1024, 16, 16, 8, 8, 1> {};
template <> struct Cfg<2048> : CfgT<2048, 16, 16, 16, 8, 1> {};
template <> struct Cfg<4096> : CfgT<4096, 16, 16, 16, 16, 1> {};
template <> struct Cfg<8192> : CfgT<8192, 16, 16, 8, 8, 8> {};

// ---------------------------------------------------------------------------------------------
// complex helpers
// ---------------------------------------------------------------------------------------------
// Packed FP32x2 arithmetic on (re, im) pairs: one FMUL2 + one FFMA2 per complex product; the swap
// and the per-half sign are operand modifiers in SASS (.F32x2.LO_HI, .NP / .PN, .F32 broadcast).
__device__ __forceinline__ float2 cmul(float2 a, float2 b)
{
    const float2 p = __fmul2_rn(a, make_float2(b.x, b.x));
    return __ffma2_rn(make_float2(a.y, a.x), make_float2(-b.y, b.y), p);
}
// a * conj(b)
__device__ __forceinline__ float2 cmulc(float2 a, float2 b)
{
    const float2 p = __fmul2_rn(a, make_float2(b.x, b.x));
    return __ffma2_rn(make_float2(a.y, a.x), make_float2(b.y, -b.y), p);
}

// In-register DFT of R points, natural order in and out.  INV = conjugate twiddles (unnormalised).
// The bodies are generated (gen_butterflies.py) in packed FP32x2 form.
template <int R, bool INV> struct Dft;
template <bool INV> struct Dft<1, INV> { __device__ __forceinline__ static void run(float2 *) {} };
#define FDAS_DFT_SPEC(R)                                                                                   \
    template <bool INV> struct Dft<R, INV> {                                                               \
        __device__ __forceinline__ static void run(float2 *v) { if (INV) dft##R##_inv(v); else dft##R##_fwd(v); } \
    };
FDAS_DFT_SPEC(2)
FDAS_DFT_SPEC(4)
FDAS_DFT_SPEC(8)
FDAS_DFT_SPEC(16)
#undef FDAS_DFT_SPEC

// ---------------------------------------------------------------------------------------------
// layouts
// ---------------------------------------------------------------------------------------------
// shared-memory address (complex elements) of (layout I, other-index o = t, digit d = 0)
template <class C, int I> __device__ __forceinline__ int lay_base(int t)
{
    constexpr int LoI = C::Lo(I);
    int lo = t % LoI, hi = t / LoI;
    int a = 0;
#pragma unroll
    for (int j = C::P - 1; j > I; --j) { a += (lo % C::R(j)) * C::stride(j); lo /= C::R(j); }
#pragma unroll
    for (int j = I - 1; j >= 1; --j) { a += (hi % C::R(j)) * C::stride(j); hi /= C::R(j); }
    if (I >= 1) a += hi * C::stride(0);
    return a;
}
// offset of (b, d) relative to lay_base in layout I
template <class C, int I> __host__ __device__ constexpr int lay_off(int b, int d)
{
    return (I == 0 ? 0 : b * C::R(I) * C::stride(0)) + d * C::stride(I);
}
// index into the w_L table of the twiddle w_{R_I Lo_I}^{d*low} = w_L^{d*low*L/(R_I Lo_I)} (per unit d)
template <class C, int I> __device__ __forceinline__ int tw_unit(int t)
{
    constexpr int LoI = C::Lo(I);
    return (t % LoI) * (C::L / (C::R(I) * LoI));
}
// natural frequency index of register (b, d) in layout P-1
template <class C> __device__ __forceinline__ int nat_freq(int t, int b, int d)
{
    int o = t + b * C::NT;
    int f = 0, w = C::L / C::R(C::P - 1);
    f += d * w;
#pragma unroll
    for (int j = C::P - 2; j >= 0; --j) {
        w /= C::R(j);
        f += (o % C::R(j)) * w;
        o /= C::R(j);
    }
    return f;
}

template <class C, int I> __device__ __forceinline__ void sm_write(float2 *buf, int base, const float2 *v)
{
    constexpr int R = C::R(I), B = C::E / R;
#pragma unroll
    for (int b = 0; b < B; ++b)
#pragma unroll
        for (int d = 0; d < R; ++d) buf[base + lay_off<C, I>(b, d)] = v[b * R + d];
}
template <class C, int I> __device__ __forceinline__ void sm_read(const float2 *buf, int base, float2 *v)
{
    constexpr int R = C::R(I), B = C::E / R;
#pragma unroll
    for (int b = 0; b < B; ++b)
#pragma unroll
        for (int d = 0; d < R; ++d) v[b * R + d] = buf[base + lay_off<C, I>(b, d)];
}
template <class C, int I, bool INV> __device__ __forceinline__ void butterflies(float2 *v)
{
    constexpr int R = C::R(I), B = C::E / R;
#pragma unroll
    for (int b = 0; b < B; ++b) Dft<R, INV>::run(v + b * R);
}

// Forward passes I..P-1 (recursive over compile-time I).  v enters in layout I (already loaded).
// bufs: two exchange buffers used alternately.  Ends in layout P-1.  Barriers: one before each
// write (WAR on the buffer pair is covered by the caller for the first write) and one after.
template <class C, int I> __device__ __forceinline__ void fwd_from(float2 *v, float2 *buf0, float2 *buf1,
                                                                   const float2 *__restrict__ tw, int t)
{
    butterflies<C, I, false>(v);
    if constexpr (I < C::P - 1) {
        constexpr int R = C::R(I), B = C::E / R;
        const int u = tw_unit<C, I>(t);
#pragma unroll
        for (int d = 1; d < R; ++d) {
            const float2 w = __ldg(tw + d * u);
#pragma unroll
            for (int b = 0; b < B; ++b) v[b * R + d] = cmul(v[b * R + d], w);
        }
        float2 *buf = (I & 1) ? buf1 : buf0;
        sm_write<C, I>(buf, lay_base<C, I>(t), v);
        __syncthreads();
        sm_read<C, I + 1>(buf, lay_base<C, I + 1>(t), v);
        fwd_from<C, I + 1>(v, buf0, buf1, tw, t);
    }
}

} // namespace fdas

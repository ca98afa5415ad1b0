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
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(float2 a, float2 b)
{
    return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
// a * conj(b)
__device__ __forceinline__ float2 cmulc(float2 a, float2 b)
{
    return make_float2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}
// multiply by -i (forward quarter turn) or +i (inverse)
template <bool INV> __device__ __forceinline__ float2 rot90(float2 a)
{
    return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
}

// cos(2 pi k / 32), k = 0..8 (double-rounded literals); other angles by symmetry at compile time.
__host__ __device__ constexpr float cos32(int k)
{
    // k in [0, 32)
    k &= 31;
    if (k > 16) k = 32 - k;          // cos is even about pi
    bool neg = false;
    if (k > 8) { k = 16 - k; neg = true; }
    float c = k == 0 ? 1.0f
            : k == 1 ? 0.98078528040323044913f
            : k == 2 ? 0.92387953251128675613f
            : k == 3 ? 0.83146961230254523708f
            : k == 4 ? 0.70710678118654752440f
            : k == 5 ? 0.55557023301960222474f
            : k == 6 ? 0.38268343236508977173f
            : k == 7 ? 0.19509032201612826785f
            : 0.0f;
    return neg ? -c : c;
}
__host__ __device__ constexpr float sin32(int k) { return cos32(k - 8); }

// v * w_R^j (forward) or v * conj(w_R^j) (inverse), R <= 32, j compile-time.
template <int R, int J, bool INV> __device__ __forceinline__ float2 mul_wconst(float2 v)
{
    constexpr int k = ((J * (32 / R)) % 32 + 32) % 32; // angle in 32nds of a turn
    if constexpr (k == 0) return v;
    else if constexpr (k == 8) return rot90<INV>(v);
    else if constexpr (k == 16) return make_float2(-v.x, -v.y);
    else if constexpr (k == 24) return rot90<!INV>(v);
    else {
        constexpr float c = cos32(k);
        constexpr float s = INV ? sin32(k) : -sin32(k); // w = c + i s with s = -sin for the forward sign
        return make_float2(v.x * c - v.y * s, v.x * s + v.y * c);
    }
}

// In-register DFT of R points, natural order in and out.  INV = conjugate twiddles (unnormalised).
template <int R, bool INV> struct Dft;
template <bool INV> struct Dft<1, INV> { __device__ __forceinline__ static void run(float2 *) {} };
template <bool INV> struct Dft<2, INV> {
    __device__ __forceinline__ static void run(float2 *v)
    {
        float2 a = cadd(v[0], v[1]), b = csub(v[0], v[1]);
        v[0] = a; v[1] = b;
    }
};
template <bool INV> struct Dft<4, INV> {
    __device__ __forceinline__ static void run(float2 *v)
    {
        float2 a0 = cadd(v[0], v[2]), a1 = csub(v[0], v[2]);
        float2 a2 = cadd(v[1], v[3]), a3 = rot90<INV>(csub(v[1], v[3]));
        v[0] = cadd(a0, a2); v[2] = csub(a0, a2);
        v[1] = cadd(a1, a3); v[3] = csub(a1, a3);
    }
};
// radix-2 split (decimation in frequency): a_j = x_j + x_{j+R/2}, b_j = (x_j - x_{j+R/2}) w_R^j,
// X_{2k} = DFT_{R/2}(a)_k, X_{2k+1} = DFT_{R/2}(b)_k.
template <int R, bool INV> struct Dft {
    template <int J> __device__ __forceinline__ static void split(float2 *v, float2 *a, float2 *b)
    {
        if constexpr (J < R / 2) {
            a[J] = cadd(v[J], v[J + R / 2]);
            b[J] = mul_wconst<R, J, INV>(csub(v[J], v[J + R / 2]));
            split<J + 1>(v, a, b);
        }
    }
    __device__ __forceinline__ static void run(float2 *v)
    {
        float2 a[R / 2], b[R / 2];
        split<0>(v, a, b);
        Dft<R / 2, INV>::run(a);
        Dft<R / 2, INV>::run(b);
#pragma unroll
        for (int k = 0; k < R / 2; ++k) { v[2 * k] = a[k]; v[2 * k + 1] = b[k]; }
    }
};

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

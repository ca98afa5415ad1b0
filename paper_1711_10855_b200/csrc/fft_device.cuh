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
// N = 1024 with 8 elements per thread (forward passes only: the stand-alone FFT of P:46, Table 1, whose design
// axis is the number of elements per thread; the convolution kernel uses Cfg<1024> with 16)
struct Cfg1024E8 : CfgT<1024, 8, 8, 8, 8, 2> {};

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

// Register part of forward pass I: butterflies of digit I, then the twiddles w_{R_I Lo_I}^{k_I low}.
template <class C, int I> __device__ __forceinline__ void fwd_pass_regs(float2 *v, const float2 *__restrict__ tw, int t)
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
    }
}

// Forward passes I..P-1 (recursive over compile-time I).  v enters in layout I (already loaded);
// REGS_DONE: the caller has already run fwd_pass_regs<C, I>.  bufs: two exchange buffers used
// alternately.  Ends in layout P-1.  Barriers: one before each write (WAR on the buffer pair is
// covered by the caller for the first write) and one after.
template <class C, int I, bool REGS_DONE = false>
__device__ __forceinline__ void fwd_from(float2 *v, float2 *buf0, float2 *buf1, const float2 *__restrict__ tw, int t)
{
    if constexpr (!REGS_DONE) fwd_pass_regs<C, I>(v, tw, t);
    if constexpr (I < C::P - 1) {
        float2 *buf = (I & 1) ? buf1 : buf0;
        sm_write<C, I>(buf, lay_base<C, I>(t), v);
        __syncthreads();
        sm_read<C, I + 1>(buf, lay_base<C, I + 1>(t), v);
        fwd_from<C, I + 1>(v, buf0, buf1, tw, t);
    }
}


// =============================================================================================
// Inverse transform of the hot loop (a4): decimation in time, passes P-1 ... 0, where the exchange
// between the first two passes is done with warp shuffles inside groups of Gs lanes and only the
// remaining exchange(s) go through shared memory.
//
// Notation: Ra = R(P-1), Rb = R(P-2); a group of Gs = Ra*Rb/E consecutive threads owns the Ra*Rb
// points that share the digits k_0..k_{P-3}; NB = E/Ra sub-transforms per thread in pass P-1,
// NA = E/Rb in pass P-2.
//   layout P-1  thread t = g*Gs + a, register i*Ra + k   <->  frequency digits (g; k_{P-2} = a*NB + i; k_{P-1} = k)
//   layout P-2  thread t = g*Gs + c, register j*Rb + tau <->  (g; k_{P-2} = (s - tau) mod Rb; n_{P-1} = c*NA + j),
//               s = NB*c + NB - 1
// The transposition a <-> c needs lane-dependent register indices; they are made static by two
// identities of the DFT:
//   * rotating the OUTPUTS of pass P-1 by rho = NA*a is a modulation of its inputs by
//     exp(+2 pi i k rho / Ra), which is folded into the template spectra G (per thread, off line);
//   * presenting the INPUTS of pass P-2 reflected and rotated, x'[tau] = x[(s - tau) mod Rb], yields
//     X'[kappa] = exp(2 pi i s kappa / Rb) X[-kappa]: a static index reflection and a unit phase
//     that is constant over each later sub-transform and therefore vanishes in |.|^2.
// In round r a thread sends registers {i*Ra + NA*r + j} to the lane r places up in its group and
// receives into {j*Rb + NB*r + NB-1-i}: 2*(Gs-1)*NA*NB 32-bit shuffles, no barrier, no bank
// conflicts, half the data-pipe wavefronts of a shared-memory exchange.
// =============================================================================================
template <class C> struct InvCfg {
    static constexpr int P = C::P, E = C::E, NT = C::NT, L = C::L;
    static constexpr int Ra = C::R(P - 1), Rb = C::R(P - 2);
    static constexpr int Gs = Ra * Rb / E, NA = E / Rb, NB = E / Ra;
    static constexpr int Q = Ra * Rb;                       // points per group
    // A half-warp spans 16/Gs groups.  Within a row of the exchange buffer the low index n_{P-1} = c*NA + j is stored
    // at lo_pos = j*Gs + c, so that the Gs threads of a group write Gs CONSECUTIVE elements per store; padding every
    // row by Gs elements then puts the groups of a half-warp on disjoint banks (64-bit accesses: 16 bank pairs).
    static constexpr int PAD = Gs >= 16 ? 0 : Gs;
    __host__ __device__ static constexpr int lo_pos(int n_lo) { return (n_lo % NA) * Gs + n_lo / NA; }
    // P == 3: one exchange, element (k_0, n_1, n_2) at k_0*STR0 + n_1*Ra + lo_pos(n_2)
    // P == 4: exchange A, element (k_0, k_1, n_2, n_3) at (k_0*R1 + k_1)*STRX + n_2*Ra + lo_pos(n_3),
    //         exchange B, element (k_0, n_1, n_2, n_3) at k_0*NT + n_1*Q + n_2*Ra + n_3
    static constexpr int STR0 = (P == 3) ? NT + PAD : NT;
    static constexpr int STRX = Q + PAD;
    static constexpr int KK = NT / Q;                       // P == 4: values of k_0 per sub-transform slot
    static constexpr int BUF_A = (P == 3) ? STR0 * C::R(0) : C::R(0) * C::R(1) * STRX;
    static constexpr int BUF_B = (P == 3) ? STR0 * C::R(0) : L;
    static constexpr int cmax(int a, int b) { return a > b ? a : b; }
    static constexpr int BUF_ELEMS = cmax(cmax(BUF_A, BUF_B), cmax(C::SMEM_ELEMS, L)); // one of the two buffers
    // register maps of the shuffle exchange (round r, sub-transforms i of pass P-1 and j of pass P-2)
    __host__ __device__ static constexpr int shfl_src_reg(int r, int i, int j) { return i * Ra + NA * r + j; }
    __host__ __device__ static constexpr int shfl_dst_reg(int r, int i, int j) { return j * Rb + NB * r + NB - 1 - i; }
    // shared-memory offsets relative to InvAddr (complex elements)
    __host__ __device__ static constexpr int wa_off(int j, int kap) { return ((Rb - kap) % Rb) * Ra + j * Gs; } // register j*Rb+kap
    __host__ __device__ static constexpr int ra_off(int b, int k) { return P == 3 ? k * STR0 : (b * KK * C::R(1) + k) * STRX; }
    __host__ __device__ static constexpr int wb_off(int b, int n) { return KK * b * STR0 + n * Q; }         // P == 4 only
    __host__ __device__ static constexpr int rb_off(int k) { return k * STR0; }                             // P == 4 only
    static_assert(P == 3 || P == 4, "three or four passes");
    static_assert(Gs >= 2 && Gs <= 32 && (Gs & (Gs - 1)) == 0, "group must be a power of two within a warp");
    static_assert(NA * Gs == Ra && NB * Gs == Rb, "group geometry");
};

// natural frequency index of register (i, k) of thread t in layout P-1 (new)
template <class C> __host__ __device__ __forceinline__ int inv_freq(int t, int i, int k)
{
    using I = InvCfg<C>;
    const int g = t / I::Gs, a = t % I::Gs;
    const int kb = a * I::NB + i;
    if constexpr (C::P == 3) return g + C::R(0) * (kb + C::R(1) * k);
    else return (g / C::R(1)) + C::R(0) * ((g % C::R(1)) + C::R(1) * (kb + C::R(2) * k));
}
// index into w_L of the modulation folded into G: G' = G * conj(w_L^idx) = G * exp(+2 pi i k NA a / Ra)
template <class C> __host__ __device__ __forceinline__ int inv_gmod_index(int t, int k)
{
    using I = InvCfg<C>;
    return (k * I::NA * (t % I::Gs) * (C::L / I::Ra)) % C::L;
}
// index into w_L of the pass P-2 multiplier of register (j, tau): v *= conj(w_L^idx)
template <class C> __host__ __device__ __forceinline__ int inv_twa_index(int t, int j, int tau)
{
    using I = InvCfg<C>;
    const int c = t % I::Gs, s = I::NB * c + I::NB - 1, n = I::NA * c + j;
    const int k_tau = ((s - tau) % I::Rb + I::Rb) % I::Rb, k_0 = s % I::Rb;
    const int e = (k_tau - k_0) * n * (C::L / (I::Ra * I::Rb));
    return ((e % C::L) + C::L) % C::L;
}
// index into w_L of the phase the outputs of thread t carry: true = out * w_L^idx ... (debug only)
template <class C> __host__ __device__ __forceinline__ int inv_fix_index(int t)
{
    using I = InvCfg<C>;
    const int q = t % I::Q, n_hi = q / I::Ra, n_lo = q % I::Ra;
    const int c = n_lo / I::NA, kap = (I::Rb - n_hi) % I::Rb, s = I::NB * c + I::NB - 1;
    // out * exp(-2 pi i s kap / Rb + 2 pi i (s mod Rb) n_lo / (Rb Ra)) = out * w_L^{s kap L/Rb - (s%Rb) n_lo L/(Ra Rb)}
    const long long e = (long long)s * kap * (C::L / I::Rb) - (long long)(s % I::Rb) * n_lo * (C::L / (I::Ra * I::Rb));
    return (int)(((e % C::L) + C::L) % C::L);
}

// 64-bit shared-memory store written as PTX so that the data operands are the producing
// instruction's own register pair (the C++ struct copy made ptxas stage every store through one
// scratch pair, a MOV/MOV/STS chain serialised by the store's read scoreboard).
__device__ __forceinline__ void st_shared_f2(float2 *p, float2 v)
{
    asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"((unsigned)__cvta_generic_to_shared(p)), "f"(v.x), "f"(v.y) : "memory");
}

// the shuffle exchange: v in layout P-1 (pass P-1 done, outputs rotated), w in layout P-2
template <class C> __device__ __forceinline__ void inv_shuffle(const float2 *v, float2 *w, int lane)
{
    using I = InvCfg<C>;
#pragma unroll
    for (int r = 0; r < I::Gs; ++r) {
        const int src = lane + (I::Gs - r); // taken modulo the group width by the hardware
#pragma unroll
        for (int i = 0; i < I::NB; ++i)
#pragma unroll
            for (int j = 0; j < I::NA; ++j) {
                float2 x = v[I::shfl_src_reg(r, i, j)];
                if (r) {
                    x.x = __shfl_sync(0xffffffffu, x.x, src, I::Gs);
                    x.y = __shfl_sync(0xffffffffu, x.y, src, I::Gs);
                }
                w[I::shfl_dst_reg(r, i, j)] = x;
            }
    }
}

// shared-memory addresses of the remaining exchange(s)
template <class C> struct InvAddr { int wa, ra, wb, rb; };
template <class C> __host__ __device__ __forceinline__ InvAddr<C> inv_addr(int t)
{
    using I = InvCfg<C>;
    InvAddr<C> A;
    // thread t reads the element whose low index is t % Ra, stored at lo_pos(t % Ra) of its Ra-block
    const int rd = t - (t % I::Ra) + I::lo_pos(t % I::Ra);
    if constexpr (C::P == 3) {
        A.wa = (t / I::Gs) * I::STR0 + (t % I::Gs);
        A.ra = rd;
        A.wb = A.rb = 0;
    } else {
        A.wa = (t / I::Gs) * I::STRX + (t % I::Gs);
        A.ra = (t / I::Q) * C::R(1) * I::STRX + (rd % I::Q);
        A.wb = (t / I::Q) * I::STR0 + (t % I::Q);
        A.rb = t;
    }
    return A;
}
// write of layout P-2 registers (pass P-2 done): register j*Rb + kappa holds n_{P-2} = (-kappa) mod Rb
template <class C> __device__ __forceinline__ void inv_write_a(float2 *buf, int wa, const float2 *w)
{
    using I = InvCfg<C>;
#pragma unroll
    for (int j = 0; j < I::NA; ++j)
#pragma unroll
        for (int kap = 0; kap < I::Rb; ++kap) st_shared_f2(buf + wa + I::wa_off(j, kap), w[j * I::Rb + kap]);
}

} // namespace fdas

// convolve.cuh -- the FDAS hot kernel (steps a1..a6 of DESIGN.md) for sm_100a.
//
// A persistent wave of CTAs; each takes (batch item, segment) work items one after the other and loops over
// all n_z templates of the item ("for every matched filter": multiply, inverse FFT, store).  Where the
// loop-invariant data live:
//   * the forward-transformed segment X and the per-thread inverse twiddles of the passes after the
//     first live in TENSOR MEMORY (tcgen05.st once per segment, tcgen05.ld per z): TMEM is a 256 KB
//     per-SM array with its own data path (measured 930 B/clk/SM), so these reads cost neither
//     registers nor LSU / shared-memory bandwidth;
//   * G_z is brought from L2 into shared memory by the bulk-copy engine (cp.async.bulk, one elected
//     thread, mbarrier completion) one z ahead and read with conflict-free LDS.128;
//   * only the working set v and addressing stay in registers (<= 128 registers, two 256-thread CTAs
//     per SM at L = 4096; the 64-thread plans L = 512, 1024 keep the pass-0 twiddles in registers too).
// The inverse transform (fft_device.cuh, "Inverse transform of the hot loop") exchanges data once
// by warp shuffles and once (L = 8192: twice) through shared memory; one barrier per exchange.
// The z loop is software pipelined: stage A of template z+1 runs before the barrier of template z.
// The same kernel has three outputs (power plane, complex plane, fused block maxima) and a variant for
// symmetric template banks.  Measured cost model, ablations and the experiments that did not help:
// profiles/r1_c3_v4.md, profiles/r2_c3_k6.md, profiles/r2_c3_k7.md.
#pragma once
#include <type_traits>

#include "fft_device.cuh"
#include "sm100_ptx.cuh"

namespace fdas {

// ---------------------------------------------------------------------------------------------
// The inverse transform in three stages (passes P-1 ... 0; fft_device.cuh "Inverse transform of the
// hot loop").  TW supplies the multipliers of pass P-2 (E entries, entry j*Rb is unused) and, for
// P == 4, of pass 1; tw0 holds w_L^{d t} for pass 0.  All multipliers are applied conjugated.
//   stage A  (in the caller) template multiply, then inv_stage_a: butterflies of pass P-1
//   stage B  shuffle exchange, multipliers, butterflies of pass P-2, write to shared memory
//   -- block barrier (the caller's: it may put independent work of the next z in front of it) --
//   stage C  read, [P == 4: pass 1 and a second exchange with its own barrier,] pass 0
// P == 3: bufa alternates between calls so that one barrier per transform suffices.
// ---------------------------------------------------------------------------------------------
template <class C> __device__ __forceinline__ void inv_stage_a(float2 *v)
{
    using I = InvCfg<C>;
#pragma unroll
    for (int i = 0; i < I::NB; ++i) Dft<I::Ra, true>::run(v + i * I::Ra);
}

template <class C, class TW>
__device__ __forceinline__ void inv_stage_b(const float2 *v, float2 *bufa, const InvAddr<C> &A, TW &tws, int lane)
{
    using I = InvCfg<C>;
    constexpr int E = C::E;
    float2 twa[E];
    tws.issue_a(twa);
    float2 w[E];
    inv_shuffle<C>(v, w, lane);
    tws.wait_a(twa);
#pragma unroll
    for (int j = 0; j < I::NA; ++j)
#pragma unroll
        for (int tau = 1; tau < I::Rb; ++tau) w[j * I::Rb + tau] = cmulc(w[j * I::Rb + tau], twa[j * I::Rb + tau]);
#pragma unroll
    for (int j = 0; j < I::NA; ++j) Dft<I::Rb, true>::run(w + j * I::Rb);
    inv_write_a<C>(bufa, A.wa, w);
}

template <class C, class TW>
__device__ __forceinline__ void inv_stage_c(float2 *v, const float2 *bufa, float2 *bufb, const InvAddr<C> &A, const float2 *tw0, TW &tws)
{
    using I = InvCfg<C>;
    constexpr int E = C::E;
    float2 tw0t[C::R(0)];
    if constexpr (TW::TW0_PARKED && C::P == 3) tws.issue_0(tw0t);
    if constexpr (C::P == 3) {
#pragma unroll
        for (int k = 0; k < C::R(0); ++k) v[k] = bufa[A.ra + I::ra_off(0, k)];
    } else {
        constexpr int R1 = C::R(1), B1 = E / R1;
        float2 twm[8];
        tws.issue_m(twm);
#pragma unroll
        for (int b = 0; b < B1; ++b)
#pragma unroll
            for (int k = 0; k < R1; ++k) v[b * R1 + k] = bufa[A.ra + I::ra_off(b, k)];
        tws.wait_m(twm);
#pragma unroll
        for (int d = 1; d < R1; ++d)
#pragma unroll
            for (int b = 0; b < B1; ++b) v[b * R1 + d] = cmulc(v[b * R1 + d], twm[d]);
#pragma unroll
        for (int b = 0; b < B1; ++b) Dft<R1, true>::run(v + b * R1);
#pragma unroll
        for (int b = 0; b < B1; ++b)
#pragma unroll
            for (int n = 0; n < R1; ++n) st_shared_f2(bufb + A.wb + I::wb_off(b, n), v[b * R1 + n]);
        if constexpr (TW::TW0_PARKED) tws.issue_0(tw0t);
        __syncthreads();
#pragma unroll
        for (int k = 0; k < C::R(0); ++k) v[k] = bufb[A.rb + I::rb_off(k)];
    }
    if constexpr (TW::TW0_PARKED) {
        tws.wait_0(tw0t);
#pragma unroll
        for (int d = 1; d < C::R(0); ++d) v[d] = cmulc(v[d], tw0t[d]);
    } else {
#pragma unroll
        for (int d = 1; d < C::R(0); ++d) v[d] = cmulc(v[d], tw0[d]);
    }
    Dft<C::R(0), true>::run(v);
}

// multipliers read from the w_L table in global memory (set-up code, debug kernel)
template <class C> struct TwLdg {
    static constexpr bool TW0_PARKED = false;
    const float2 *__restrict__ tw;
    int t;
    __device__ __forceinline__ void issue_a(float2 *o) const
    {
        using I = InvCfg<C>;
#pragma unroll
        for (int j = 0; j < I::NA; ++j) {
            o[j * I::Rb] = make_float2(1.f, 0.f);
#pragma unroll
            for (int tau = 1; tau < I::Rb; ++tau) o[j * I::Rb + tau] = __ldg(tw + inv_twa_index<C>(t, j, tau));
        }
    }
    __device__ __forceinline__ void wait_a(float2 *) const {}
    __device__ __forceinline__ void issue_m(float2 *o) const
    {
        if constexpr (C::P == 4) {
            const int u = tw_unit<C, 1>(t);
            o[0] = make_float2(1.f, 0.f);
#pragma unroll
            for (int d = 1; d < C::R(1); ++d) o[d] = __ldg(tw + d * u);
        }
    }
    __device__ __forceinline__ void wait_m(float2 *) const {}
};

// tensor-memory geometry: per thread (TMEM lane) a block of columns X | TWA [| TWM]
template <class C> struct TmemCfg {
    static constexpr int SLOTS = (C::NT + 127) / 128;          // warps sharing a 32-lane quarter
    static constexpr int X_OFF = 0, TWA_OFF = 32, TW0_OFF = 64, TWM_OFF = 96;
    static constexpr bool TW0_PARKED = C::NT >= 128;           // pass-0 multipliers in TMEM too (else registers)
    static constexpr int SLOT_COLS = TW0_PARKED ? 128 : 64;
    static constexpr int NCOLS_RAW = SLOT_COLS * SLOTS;
    static constexpr int NCOLS = NCOLS_RAW <= 32 ? 32 : NCOLS_RAW <= 64 ? 64 : NCOLS_RAW <= 128 ? 128 : NCOLS_RAW <= 256 ? 256 : 512;
    static constexpr int MINB = (512 / C::NT) > 0 ? (512 / C::NT) : 1; // CTAs per SM at 128 registers
    static_assert(2 * C::E <= 32, "a segment slice or a twiddle block is at most 32 columns");
    static_assert(NCOLS_RAW <= 512 && NCOLS * MINB <= 512, "tensor memory holds 512 columns per SM");
    static_assert(TW0_PARKED || C::P == 3, "four passes need the 128-column block");
};

// multipliers parked in tensor memory
template <class C> struct TwTmem {
    static constexpr bool TW0_PARKED = TmemCfg<C>::TW0_PARKED;
    uint32_t addr; // TMEM address of this thread's column block
    __device__ __forceinline__ void issue_0(float2 *o) const
    {
        ptx::tmem_ld16(addr + TmemCfg<C>::TW0_OFF, o);
        if constexpr (C::R(0) > 8) ptx::tmem_ld16(addr + TmemCfg<C>::TW0_OFF + 16, o + 8);
    }
    __device__ __forceinline__ void wait_0(float2 *o) const
    {
        ptx::tmem_wait_ld8(o);
        if constexpr (C::R(0) > 8) ptx::tmem_wait_ld8(o + 8);
    }
    __device__ __forceinline__ void issue_a(float2 *o) const
    {
        ptx::tmem_ld16(addr + TmemCfg<C>::TWA_OFF, o);
        if constexpr (C::E > 8) ptx::tmem_ld16(addr + TmemCfg<C>::TWA_OFF + 16, o + 8);
    }
    __device__ __forceinline__ void wait_a(float2 *o) const
    {
        ptx::tmem_wait_ld8(o);
        if constexpr (C::E > 8) ptx::tmem_wait_ld8(o + 8);
    }
    __device__ __forceinline__ void issue_m(float2 *o) const
    {
        if constexpr (C::P == 4) ptx::tmem_ld16(addr + TmemCfg<C>::TWM_OFF, o);
    }
    __device__ __forceinline__ void wait_m(float2 *o) const
    {
        if constexpr (C::P == 4) ptx::tmem_wait_ld8(o);
    }
};

// forward transform of v (natural order, v[d] = x[d*NT + t]) into layout P-1 of the inverse:
// the decimation-in-frequency passes of fft_device.cuh followed by one re-layout through buf0.
// REGS_DONE: the caller has already run fwd_pass_regs<C, 0> on v.
template <class C, bool REGS_DONE = false>
__device__ __forceinline__ void forward_to_inv_layout(float2 *v, float2 *buf0, float2 *buf1, const float2 *__restrict__ tw, int t)
{
    using I = InvCfg<C>;
    constexpr int RL = C::R(C::P - 1), BL = C::E / RL;
    fwd_from<C, 0, REGS_DONE>(v, buf0, buf1, tw, t);
    __syncthreads();
    // element of natural frequency f sits at f + f/16: both index maps step through f in strides of 16
    // within a half-warp, which the extra element per 16 spreads over the banks
    static_assert(I::BUF_ELEMS >= C::L + C::L / 16, "re-layout buffer");
#pragma unroll
    for (int b = 0; b < BL; ++b)
#pragma unroll
        for (int d = 0; d < RL; ++d) {
            const int f = nat_freq<C>(t, b, d);
            buf0[f + (f >> 4)] = v[b * RL + d];
        }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < I::NB; ++i)
#pragma unroll
        for (int k = 0; k < I::Ra; ++k) {
            const int f = inv_freq<C>(t, i, k);
            v[i * I::Ra + k] = buf0[f + (f >> 4)];
        }
}

// |y|^2 (a5) with the rounding spelled out, so that every output mode produces the same bits
__device__ __forceinline__ float power_of(float2 y) { return __fmaf_rn(y.x, y.x, __fmul_rn(y.y, y.y)); }

struct ConvParams {
    const float2 *__restrict__ spectrum; // [n_batch][n_f]
    float *__restrict__ power;           // OUT_POWER: [n_batch][n_z][n_f]
    float2 *__restrict__ amp;            // OUT_AMP: [n_batch][n_z][n_f] complex A' (eq.(2) itself)
    float *__restrict__ bmax;            // OUT_BLOCKMAX: [n_batch][n_z][n_seg] maximum power of the segment's columns
    int *__restrict__ barg;              // OUT_BLOCKMAX: [n_batch][n_z][n_seg] lowest column offset attaining it
    const float4 *__restrict__ gperm;    // [n_z][E/2][NT] : template spectra in register order
    const float2 *__restrict__ tw;       // [L] : w_L^j
    unsigned int *__restrict__ work;     // [2] : next work item, CTAs finished (both 0 between launches)
    int64_t n_f;
    int64_t n_seg;
    int64_t n_work;                      // one past the last work item of this launch (n_batch * n_seg for a whole call)
    int64_t w_begin;                     // first work item of this launch (0 for a whole call)
    int n_z;
    int m;
    int S;
    int bulk_ok;                         // spectrum base is 16-byte aligned: interior segments may be bulk-copied
};

// What the kernel does with the filtered segment y_z (a5, a6):
//   OUT_POWER     |y|^2 -> float32 power plane (BASELINE.json north_star)
//   OUT_AMP       y itself -> complex64 plane: the paper's general convolution (Table 2)
//   OUT_BLOCKMAX  max and argmax of |y|^2 over the segment's S columns: the plane never reaches HBM
//                 (reading 17)
enum { OUT_POWER = 0, OUT_AMP = 1, OUT_BLOCKMAX = 2 };

template <class C> constexpr size_t conv_smem_bytes()
{
    return 2 * sizeof(float2) * (size_t)InvCfg<C>::BUF_ELEMS + sizeof(float2) * (size_t)C::L;
}

// Persistent kernel: the grid is one wave of resident CTAs (fdas.cu sizes it from the occupancy and
// the tensor-memory budget); every CTA sets up its tensor-memory tables once and then takes
// (batch item, segment) work items from a global counter until none is left.  Dynamic rather than
// strided assignment because the CTAs sharing an SM do not run at the same speed (profiles/r1_c3_v5.md).
// SYM ("FDAS specific ... symmetries"): the bank satisfies h_{-z} = conj(h_{+z})
// (checked by fdas_set_templates).  Then P[-z](A) = P[+z](conj A) exactly, i.e. row -z is the same template
// applied to DFT(conj x)[n] = conj(X[-n]), which is parked in tensor memory next to X: one template fetch
// serves two rows.  The shortcut G_{-z} = conj(G_{+z}) is NOT exact for an even window and is not used.
template <int L, int OUT, bool SYM = false>
__global__ void __launch_bounds__(Cfg<L>::NT, TmemCfg<Cfg<L>>::MINB) fdas_convolve_kernel(const ConvParams p)
{
    using C = Cfg<L>;
    using I = InvCfg<C>;
    using TC = TmemCfg<C>;
    constexpr int E = C::E, NT = C::NT;
    constexpr uint32_t G_BYTES = (uint32_t)L * 8u;
    constexpr int D0_FAST = E / 8;       // first kept register when m = L/8 (every BASELINE.json config)
    constexpr int XC_OFF = TC::TWM_OFF;  // SYM: DFT(conj x) sits in the column block that four-pass plans use for twiddles
    static_assert(!SYM || (C::P == 3 && TC::TW0_PARKED && OUT == OUT_POWER), "SYM needs the free 32-column block");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float2 *buf0 = reinterpret_cast<float2 *>(smem_raw);
    float2 *buf1 = buf0 + I::BUF_ELEMS;
    float4 *gs = reinterpret_cast<float4 *>(buf1 + I::BUF_ELEMS); // [E/2][NT]: template stage / segment stage
    __shared__ __align__(8) uint64_t g_bar;
    __shared__ uint32_t tmem_slot;
    __shared__ uint32_t s_work[2];
    __shared__ uint2 s_part[2][(Cfg<L>::NT + 31) / 32]; // OUT_BLOCKMAX: per-warp (power bits, position), by parity of z

    const int t = threadIdx.x, warp = t >> 5, lane = t & 31;

    if (t == 0) {
        ptx::mbar_init(&g_bar, 1);
        ptx::mbar_fence_init();
    }
    if (warp == 0) ptx::tmem_alloc<TC::NCOLS>(&tmem_slot);
    ptx::tmem_fence_before_sync();
    __syncthreads();
    ptx::tmem_fence_after_sync();
    const uint32_t tm_addr = tmem_slot + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)(TC::SLOT_COLS * (warp >> 2));

    // inverse multipliers (independent of z and of the segment): once per CTA.  Pass 0 in
    // registers for the 64-thread plans, everything else in tensor memory.
    float2 tw0[TC::TW0_PARKED ? 1 : C::R(0)];
    {
        if constexpr (TC::TW0_PARKED) {
            float2 w0[16];
#pragma unroll
            for (int d = 0; d < 16; ++d) w0[d] = (d && d < C::R(0)) ? __ldg(p.tw + d * t) : make_float2(1.f, 0.f);
            ptx::tmem_st16(tm_addr + TC::TW0_OFF, w0);
            if constexpr (C::R(0) > 8) ptx::tmem_st16(tm_addr + TC::TW0_OFF + 16, w0 + 8);
        } else {
            tw0[0] = make_float2(1.f, 0.f);
#pragma unroll
            for (int d = 1; d < C::R(0); ++d) tw0[d] = __ldg(p.tw + d * t);
        }
        TwLdg<C> src{p.tw, t};
        float2 w[16];
#pragma unroll
        for (int d = 0; d < 16; ++d) w[d] = make_float2(1.f, 0.f);
        src.issue_a(w);
        ptx::tmem_st16(tm_addr + TC::TWA_OFF, w);
        if constexpr (E > 8) ptx::tmem_st16(tm_addr + TC::TWA_OFF + 16, w + 8);
        if constexpr (C::P == 4) {
            src.issue_m(w);
            ptx::tmem_st16(tm_addr + TC::TWM_OFF, w);
        }
    }
    const InvAddr<C> A = inv_addr<C>(t);
    TwTmem<C> tws{tm_addr};
    uint32_t gphase = 0; // parity of the next completion of g_bar
    const bool fast_m = (p.m * 8 == L);
    // OUT_AMP: the unit phase the static shuffle exchange leaves on this thread's outputs (fft_device.cuh)
    float2 fix = make_float2(1.f, 0.f);
    if constexpr (OUT == OUT_AMP) fix = __ldg(p.tw + inv_fix_index<C>(t));

    // a1 through the bulk-copy engine: segment `w` can be copied as one 16-byte aligned block of L
    // complex64 if it lies inside [0, n_f); the first and last segment(s) need the zero padding of
    // reading 6 and are loaded with guarded loads instead.
    auto seg_base = [&](uint32_t w) { return (int64_t)(w % p.n_seg) * p.S - p.m / 2; };
    auto seg_bulk = [&](uint32_t w) {
        const int64_t base = seg_base(w);
        return p.bulk_ok && base >= 0 && base + L <= p.n_f && (((w / p.n_seg) * p.n_f + base) & 1) == 0;
    };
    auto fetch_segment = [&](uint32_t w) { // elected thread
        const float2 *src = p.spectrum + (int64_t)(w / p.n_seg) * p.n_f + seg_base(w);
        ptx::mbar_expect_tx(&g_bar, G_BYTES);
        ptx::bulk_g2s(gs, src, G_BYTES, &g_bar);
    };

    // Work items: the first is the CTA's own index, the others come from the counter (which therefore counts from
    // gridDim.x).  A wave of CTAs that starts together would otherwise open with hundreds of atomics on one address.
    const uint32_t n_mine = (uint32_t)(p.n_work - p.w_begin); // items of this launch
    uint32_t w = (uint32_t)p.w_begin + blockIdx.x;
    int slot = 0;
    if (t == 0 && w < p.n_work && seg_bulk(w)) fetch_segment(w);

    while (w < p.n_work) {
        const int64_t seg = w % p.n_seg;
        const int64_t bi = w / p.n_seg;
        uint32_t w_next = 0;
        if (t == 0) // used after the next barriers
            w_next = (gridDim.x < n_mine) ? (uint32_t)p.w_begin + gridDim.x + atomicAdd(p.work, 1u) : (uint32_t)p.n_work;

        // a1: segment load, x[i] = A[seg*S - m/2 + i], zero outside [0, n_f)  (reading 6)
        float2 v[E];
        if (seg_bulk(w)) {
            ptx::mbar_wait(&g_bar, gphase);
            gphase ^= 1;
            const float2 *xs = reinterpret_cast<const float2 *>(gs);
#pragma unroll
            for (int d = 0; d < E; ++d) v[d] = xs[d * NT + t];
        } else {
            const float2 *__restrict__ Ab = p.spectrum + bi * p.n_f;
            const int64_t base = seg * p.S - p.m / 2;
#pragma unroll
            for (int d = 0; d < E; ++d) {
                const int64_t k = base + d * NT + t;
                v[d] = (k >= 0 && k < p.n_f) ? __ldg(Ab + k) : make_float2(0.f, 0.f);
            }
        }
        // a2: forward FFT, once per segment (eq.(3)); the result is parked in tensor memory.  The register
        // part of its first pass comes before the barrier that releases the stage to the bulk-copy engine:
        // the engine does not queue behind this thread's loads, so they must have returned (been used)
        // before the thread arrives.
        fwd_pass_regs<C, 0>(v, p.tw, t);
        __syncthreads(); // the stage is read; the previous item's last exchange reads are done
        if (t == 0) {    // template spectrum of z = 0 (a3), in flight during the forward transform
            ptx::mbar_expect_tx(&g_bar, G_BYTES);
            ptx::bulk_g2s(gs, p.gperm, G_BYTES, &g_bar);
        }
        forward_to_inv_layout<C, true>(v, buf0, buf1, p.tw, t);
        ptx::tmem_st16(tm_addr + TC::X_OFF, v);
        if constexpr (E > 8) ptx::tmem_st16(tm_addr + TC::X_OFF + 16, v + 8);
        if constexpr (SYM) { // DFT(conj x)[f] = conj(X[-f]) from the natural-order copy the re-layout left in buf0
            float2 xc[E];
#pragma unroll
            for (int i = 0; i < I::NB; ++i)
#pragma unroll
                for (int k = 0; k < I::Ra; ++k) {
                    const int f = (L - inv_freq<C>(t, i, k)) & (L - 1);
                    const float2 a = buf0[f + (f >> 4)];
                    xc[i * I::Ra + k] = make_float2(a.x, -a.y);
                }
            ptx::tmem_st16(tm_addr + XC_OFF, xc);
            if constexpr (E > 8) ptx::tmem_st16(tm_addr + XC_OFF + 16, xc + 8);
        }
        ptx::tmem_wait_st();

        // The z loop runs n_z iterations.  Iteration k: template G_{g(k)} on X (sel 0) or on DFT(conj x) (sel 1)
        // produces row r(k).  Without SYM g = r = k.  With SYM the rows are taken in pairs (j, n_z-1-j), j = k/2,
        // and the middle row (z = 0) alone at the end.
        const int n_g = SYM ? (p.n_z + 1) / 2 : p.n_z;                        // templates fetched per segment
        auto it_sel = [&](int k) { return SYM ? (k & 1) : 0; };
        auto it_row = [&](int k) { return SYM ? ((k & 1) ? p.n_z - 1 - (k >> 1) : (k >> 1)) : k; };
        auto it_last_use = [&](int k) { return SYM ? ((k & 1) || k == p.n_z - 1) : true; };
        int g_next = 1; // elected thread: next template to fetch

        const int64_t col0 = seg * p.S - p.m + t;                             // column of y[t]
        float *__restrict__ out = p.power + bi * p.n_z * p.n_f + col0;        // row 0 of this batch item
        float *const out0 = out;
        float2 *__restrict__ out_c = p.amp + bi * p.n_z * p.n_f + col0;
        int64_t bm_idx = (bi * p.n_z) * p.n_seg + seg;                         // OUT_BLOCKMAX: entry of row 0
        const bool interior = (seg + 1) * (int64_t)p.S <= p.n_f;
        const bool fast8 = interior && fast_m;
        const bool fast = interior && (p.m % NT == 0) && (p.m / NT <= 4);
        const int d0 = p.m / NT;

        // a3 + first inverse pass of template z ("convolution in the Fourier domain"; "for every
        // matched filter"): v = X * G_z in layout P-1, butterflies of pass P-1
        auto stage_a = [&](int k) {
            float2 X[E];
            const uint32_t xa = tm_addr + (it_sel(k) ? XC_OFF : TC::X_OFF);
            ptx::tmem_ld16(xa, X);
            if constexpr (E > 8) ptx::tmem_ld16(xa + 16, X + 8);
            if (!it_sel(k)) { // a new template: wait for its bulk copy
                ptx::mbar_wait(&g_bar, gphase);
                gphase ^= 1;
            }
            ptx::tmem_wait_ld8(X);
            if constexpr (E > 8) ptx::tmem_wait_ld8(X + 8);
#pragma unroll
            for (int q = 0; q < E / 2; ++q) {
                const float4 g = gs[q * NT + t];
                v[2 * q] = cmul(X[2 * q], make_float2(g.x, g.y));
                v[2 * q + 1] = cmul(X[2 * q + 1], make_float2(g.z, g.w));
            }
            inv_stage_a<C>(v);
        };
        // elected thread, after the barrier that follows stage A of iteration k (every thread is past its reads of
        // the stage): if that was the last use of its template, fetch the next one, or after the last template the
        // next work item's segment
        auto after_stage_a = [&](int k) {
            if (t == 0 && it_last_use(k)) {
                if (g_next < n_g) {
                    ptx::mbar_expect_tx(&g_bar, G_BYTES);
                    ptx::bulk_g2s(gs, reinterpret_cast<const unsigned char *>(p.gperm) + (size_t)g_next * G_BYTES, G_BYTES, &g_bar);
                } else if (g_next == n_g) { // first use of w_next: the atomic has had nearly the whole segment to return
                    s_work[slot ^ 1] = w_next;
                    if (w_next < p.n_work && seg_bulk(w_next)) fetch_segment(w_next);
                }
                ++g_next;
            }
        };
        stage_a(0);
        __syncthreads(); // also: the forward transform's last reads of buf0 are done before the z loop writes it
        after_stage_a(0);

        // The z loop is software pipelined: stage A of template z+1 (tensor-memory and shared-memory
        // reads, 1/3 of the arithmetic) sits between the exchange write of template z and its barrier, so
        // a warp that reaches the barrier early has independent work instead of idling.  The loop exists
        // once per store mode (a5 + a6 below) so that the mode costs nothing inside it.
        // OUT_BLOCKMAX: block result of template zz from the per-warp partials (one warp, after a barrier)
        auto finalize_max = [&](int zz) {
            if (warp == 0) {
                constexpr int NW = (NT + 31) / 32;
                const uint2 pr = lane < NW ? s_part[zz & 1][lane] : make_uint2(0u, 0x7fffffffu);
                const unsigned wm = __reduce_max_sync(0xffffffffu, pr.x);
                const unsigned wc = __reduce_min_sync(0xffffffffu, pr.x == wm ? pr.y : 0x7fffffffu);
                if (lane == 0) {
                    const int64_t o = bm_idx + (int64_t)zz * p.n_seg;
                    p.bmax[o] = __uint_as_float(wm);
                    p.barg[o] = (int)wc - p.m;
                }
            }
        };
        auto z_loop = [&](auto mode_tag) {
            constexpr int MODE = decltype(mode_tag)::value;
            // which registers are outputs of this segment: u[d] is y[d*NT + t], kept if m <= d*NT + t < m + S
            // and its column exists.  MODE 0: interior segment and m = L/8; MODE 1: interior segment and m a
            // small multiple of the thread count; MODE 2: anything else, per-element bounds.
            auto kept = [&](int d) -> bool {
                if constexpr (MODE == 0) return d >= D0_FAST;
                else if constexpr (MODE == 1) return d >= 4 || d >= d0;
                else {
                    const int pidx = d * NT + t;
                    return pidx >= p.m && pidx < p.m + p.S && col0 + d * NT < p.n_f;
                }
            };
            for (int z = 0; z < p.n_z; ++z) {
                float2 *bufa = (C::P == 3 && (z & 1)) ? buf1 : buf0;
                inv_stage_b<C>(v, bufa, A, tws, lane);
                if (z + 1 < p.n_z) stage_a(z + 1);
                __syncthreads();
                if (z + 1 < p.n_z) after_stage_a(z + 1);
                if constexpr (OUT == OUT_BLOCKMAX) {
                    if (z > 0) finalize_max(z - 1);
                }
                float2 u[E];
                inv_stage_c<C>(u, bufa, buf1, A, tw0, tws);
                // a5 + a6: trim, then power / amplitude / block maximum
                if constexpr (OUT == OUT_POWER) {
                    if constexpr (SYM) out = out0 + (int64_t)it_row(z) * p.n_f;
#pragma unroll
                    for (int d = 0; d < E; ++d) {
                        if (MODE == 0 && d < D0_FAST) continue;
                        if (kept(d)) {
                            const float pw = power_of(u[d]);
                            if constexpr (MODE == 2) out[d * NT] = pw;
                            else __stcs(out + d * NT, pw);
                        }
                    }
                    if constexpr (!SYM) out += p.n_f;
                } else if constexpr (OUT == OUT_AMP) {
#pragma unroll
                    for (int d = 0; d < E; ++d) {
                        if (MODE == 0 && d < D0_FAST) continue;
                        if (kept(d)) {
                            const float2 a = cmul(u[d], fix);
                            if constexpr (MODE == 2) out_c[d * NT] = a;
                            else __stcs(out_c + d * NT, a);
                        }
                    }
                    out_c += p.n_f;
                } else {
                    float pw[E];
                    float best = 0.f; // powers are >= 0, so their bit patterns order like unsigned integers
#pragma unroll
                    for (int d = 0; d < E; ++d) {
                        pw[d] = power_of(u[d]);
                        if (MODE == 0 && d < D0_FAST) continue;
                        if (kept(d)) best = fmaxf(best, pw[d]);
                    }
                    const unsigned wm = __reduce_max_sync(0xffffffffu, __float_as_uint(best));
                    unsigned pos = 0x7fffffffu;
                    if (__float_as_uint(best) == wm) { // rare: the lanes that hold the warp's maximum look up where
#pragma unroll
                        for (int d = E - 1; d >= 0; --d) {
                            if (MODE == 0 && d < D0_FAST) continue;
                            if (kept(d) && __float_as_uint(pw[d]) == wm) pos = (unsigned)(d * NT + t);
                        }
                    }
                    const unsigned wp = __reduce_min_sync(0xffffffffu, pos);
                    if (lane == 0) s_part[z & 1][warp] = make_uint2(wm, wp);
                }
            }
        };
        if (fast8) z_loop(std::integral_constant<int, 0>{});
        else if (fast) z_loop(std::integral_constant<int, 1>{});
        else z_loop(std::integral_constant<int, 2>{});
        if constexpr (OUT == OUT_BLOCKMAX) {
            __syncthreads();
            finalize_max(p.n_z - 1);
        }
        slot ^= 1;
        w = s_work[slot];
    }
    ptx::tmem_fence_before_sync();
    __syncthreads();
    if (warp == 0) ptx::tmem_free<TC::NCOLS>(tmem_slot);
    if (t == 0 && gridDim.x < n_mine) { // the last CTA out re-arms the counters for the next launch
        __threadfence();
        if (atomicAdd(p.work + 1, 1u) == gridDim.x - 1) {
            p.work[0] = 0;
            p.work[1] = 0;
            __threadfence();
        }
    }
}

} // namespace fdas

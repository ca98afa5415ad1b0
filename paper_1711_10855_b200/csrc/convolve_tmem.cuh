// convolve_tmem.cuh -- the FDAS hot kernel, occupancy-first variant for sm_100a.
//
// Same arithmetic and the same layouts as fdas_convolve_kernel (fdas.cu); what changes is where the
// loop-invariant data live.  The z loop of P:46 ("for every matched filter": multiply, inverse FFT,
// store) needs, per thread, the forward-transformed segment X (2E words), the inverse twiddles of
// every pass (up to 60 words) and the incoming template spectrum G_z (2E words).  Held in registers
// that is 186 registers and one 8-warp CTA per SM, and ncu shows the kernel latency bound
// (profiles/r1_c3_v1.md).  Here
//   * X and the twiddles of passes >= 1 live in TENSOR MEMORY (tcgen05.st once per segment,
//     tcgen05.ld per z): TMEM is a 256 KB per-SM array with its own data path, so these reads cost
//     neither registers nor LSU / shared-memory bandwidth (measured: >= 320 B/clk/SM, concurrent with LDS),
//   * G_z is brought from L2 into shared memory by the bulk-copy engine (cp.async.bulk, one elected
//     thread, mbarrier completion) one z ahead, and read with conflict-free LDS.128 when it is used,
//   * only the working set v, the pass-0 twiddles and addressing stay in registers: <= 128 registers,
//     so twice the warps are resident and one CTA's exchange phase overlaps another's butterflies.
#pragma once
#include "fft_device.cuh"
#include "sm100_ptx.cuh"

namespace fdas {

template <class C> struct TmemCfg {
    static constexpr int SLOTS = (C::NT + 127) / 128;          // warps sharing a 32-lane quarter
    static constexpr int XW = 32;                              // column stride of one slot (>= 2E)
    static constexpr int X_COL0 = 0;
    static constexpr int TW_COL0 = XW * SLOTS;
    static constexpr int NCOLS_RAW = 2 * XW * SLOTS;
    static constexpr int NCOLS = NCOLS_RAW <= 32 ? 32 : NCOLS_RAW <= 64 ? 64 : NCOLS_RAW <= 128 ? 128 : NCOLS_RAW <= 256 ? 256 : 512;
    static constexpr int MINB = (512 / C::NT) > 0 ? (512 / C::NT) : 1; // CTAs per SM at 128 registers
    // twiddles of pass I >= 1 sit at complex slots [tw_slot(I), tw_slot(I) + R(I)) of a 16-slot block
    __host__ __device__ static constexpr int tw_slot(int I) { return I == 1 ? 0 : 8; }
    static_assert(C::P == 3 || (C::R(1) <= 8 && C::R(2) <= 8), "twiddle block holds 16 complex values");
    static_assert(2 * C::E <= XW, "segment does not fit its TMEM slot");
};

struct TmemCtx {
    uint32_t x_addr;   // TMEM address of this thread's X row
    uint32_t tw_addr;  // TMEM address of this thread's twiddle row
};

// Inverse passes with twiddles of pass I >= 1 fetched from TMEM while the exchange barrier is pending.
template <class C, int I, class Hook>
__device__ __forceinline__ void inv_down_tmem(float2 *v, float2 *buf0, float2 *buf1, const float2 *tw0, const TmemCtx &tm,
                                              const int *bases, Hook &&after_first_barrier)
{
    constexpr int R = C::R(I), B = C::E / R;
    float2 *buf = (I & 1) ? buf1 : buf0;
    sm_write<C, I + 1>(buf, bases[I + 1], v);
    float2 w[16];
    if constexpr (I >= 1) {
        ptx::tmem_ld16(tm.tw_addr + 2 * TmemCfg<C>::tw_slot(I), w);
        if constexpr (R > 8) ptx::tmem_ld16(tm.tw_addr + 2 * TmemCfg<C>::tw_slot(I) + 16, w + 8);
    }
    __syncthreads();
    if constexpr (I == C::P - 2) after_first_barrier();
    sm_read<C, I>(buf, bases[I], v);
    if constexpr (I >= 1) {
        ptx::tmem_wait_ld8(w);
        if constexpr (R > 8) ptx::tmem_wait_ld8(w + 8);
#pragma unroll
        for (int d = 1; d < R; ++d)
#pragma unroll
            for (int b = 0; b < B; ++b) v[b * R + d] = cmulc(v[b * R + d], w[d]);
    } else {
#pragma unroll
        for (int d = 1; d < R; ++d)
#pragma unroll
            for (int b = 0; b < B; ++b) v[b * R + d] = cmulc(v[b * R + d], tw0[d]);
    }
    butterflies<C, I, true>(v);
    if constexpr (I > 0) inv_down_tmem<C, I - 1>(v, buf0, buf1, tw0, tm, bases, after_first_barrier);
}

template <class C, int I> __device__ __forceinline__ void fill_bases_t(int *bases, int t)
{
    bases[I] = lay_base<C, I>(t);
    if constexpr (I + 1 < C::P) fill_bases_t<C, I + 1>(bases, t);
}

struct ConvParams {
    const float2 *__restrict__ spectrum; // [n_batch][n_f]
    float *__restrict__ power;           // [n_batch][n_z][n_f]
    const float4 *__restrict__ gperm;    // [n_z][E/2][NT] : template spectra in register order
    const float2 *__restrict__ tw;       // [L] : w_L^j
    int64_t n_f;
    int64_t n_seg;
    int n_z;
    int m;
    int S;
};

template <int L>
__global__ void __launch_bounds__(Cfg<L>::NT, TmemCfg<Cfg<L>>::MINB) fdas_convolve_tmem_kernel(const ConvParams p)
{
    using C = Cfg<L>;
    using TC = TmemCfg<C>;
    constexpr int E = C::E, NT = C::NT;
    constexpr uint32_t G_BYTES = (uint32_t)L * 8u;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float2 *buf0 = reinterpret_cast<float2 *>(smem_raw);
    float2 *buf1 = buf0 + C::SMEM_ELEMS;
    float4 *gs = reinterpret_cast<float4 *>(buf1 + C::SMEM_ELEMS); // [E/2][NT]
    __shared__ __align__(8) uint64_t g_bar;
    __shared__ uint32_t tmem_slot;

    const int t = threadIdx.x, warp = t >> 5;
    const int64_t seg = blockIdx.x % p.n_seg;
    const int64_t bi = blockIdx.x / p.n_seg;

    if (t == 0) {
        ptx::mbar_init(&g_bar, 1);
        ptx::mbar_fence_init();
    }
    if (warp == 0) ptx::tmem_alloc<TC::NCOLS>(&tmem_slot);
    ptx::tmem_fence_before_sync();
    __syncthreads();
    ptx::tmem_fence_after_sync();
    if (t == 0) { // template spectrum of z = 0 (a3), in flight during the forward transform
        ptx::mbar_expect_tx(&g_bar, G_BYTES);
        ptx::bulk_g2s(gs, p.gperm, G_BYTES, &g_bar);
    }
    TmemCtx tm;
    {
        const uint32_t lane_base = (uint32_t)(32 * (warp & 3)) << 16;
        const uint32_t slot = (uint32_t)(warp >> 2);
        tm.x_addr = tmem_slot + lane_base + TC::X_COL0 + TC::XW * slot;
        tm.tw_addr = tmem_slot + lane_base + TC::TW_COL0 + TC::XW * slot;
    }

    // a1: segment load, x[i] = A[seg*S - m/2 + i], zero outside [0, n_f)  (reading 6)
    float2 v[E];
    {
        const float2 *__restrict__ A = p.spectrum + bi * p.n_f;
        const int64_t base = seg * p.S - p.m / 2;
#pragma unroll
        for (int d = 0; d < E; ++d) {
            const int64_t k = base + d * NT + t;
            v[d] = (k >= 0 && k < p.n_f) ? __ldg(A + k) : make_float2(0.f, 0.f);
        }
    }
    // a2: forward FFT, once per segment (eq.(3)); the result is parked in tensor memory
    fwd_from<C, 0>(v, buf0, buf1, p.tw, t);
    ptx::tmem_st16(tm.x_addr, v);
    if constexpr (E > 8) ptx::tmem_st16(tm.x_addr + 16, v + 8);

    // inverse twiddles (independent of z): pass 0 in registers, passes >= 1 in tensor memory
    float2 tw0[C::R(0)];
    {
        const int u0 = tw_unit<C, 0>(t);
        tw0[0] = make_float2(1.f, 0.f);
#pragma unroll
        for (int d = 1; d < C::R(0); ++d) tw0[d] = __ldg(p.tw + d * u0);
        float2 w[16];
#pragma unroll
        for (int d = 0; d < 16; ++d) w[d] = make_float2(1.f, 0.f);
        const int u1 = tw_unit<C, 1>(t);
#pragma unroll
        for (int d = 1; d < C::R(1); ++d) w[TC::tw_slot(1) + d] = __ldg(p.tw + d * u1);
        if constexpr (C::P == 4) {
            const int u2 = tw_unit<C, 2>(t);
#pragma unroll
            for (int d = 1; d < C::R(2); ++d) w[TC::tw_slot(2) + d] = __ldg(p.tw + d * u2);
        }
        ptx::tmem_st16(tm.tw_addr, w);
        ptx::tmem_st16(tm.tw_addr + 16, w + 8);
    }
    ptx::tmem_wait_st();
    __syncthreads(); // forward transform's last reads of buf0/buf1 are done before the z loop writes them

    int bases[C::P];
    fill_bases_t<C, 0>(bases, t);

    const int64_t col0 = seg * p.S - p.m + t;                 // column of y[t]
    float *__restrict__ prow = p.power + bi * p.n_z * p.n_f;  // row 0 of this batch item
    const bool interior = (seg + 1) * (int64_t)p.S <= p.n_f;
    const bool fast = interior && (p.m % NT == 0) && (p.m / NT <= 4);
    const int d0 = p.m / NT;

    for (int z = 0; z < p.n_z; ++z) {
        // a3: pointwise multiply by the transformed template ("convolution in the Fourier domain")
        float2 X[E];
        ptx::tmem_ld16(tm.x_addr, X);
        if constexpr (E > 8) ptx::tmem_ld16(tm.x_addr + 16, X + 8);
        ptx::mbar_wait(&g_bar, (uint32_t)(z & 1));
        ptx::tmem_wait_ld8(X);
        if constexpr (E > 8) ptx::tmem_wait_ld8(X + 8);
#pragma unroll
        for (int q = 0; q < E / 2; ++q) {
            const float4 g = gs[q * NT + t];
            v[2 * q] = cmul(X[2 * q], make_float2(g.x, g.y));
            v[2 * q + 1] = cmul(X[2 * q + 1], make_float2(g.z, g.w));
        }
        // a4: inverse FFT; after the first exchange barrier every thread has consumed G_z, so the
        // elected thread starts the bulk copy of G_{z+1} into the same stage
        butterflies<C, C::P - 1, true>(v);
        inv_down_tmem<C, C::P - 2>(v, buf0, buf1, tw0, tm, bases, [&]() {
            if (t == 0 && z + 1 < p.n_z) {
                ptx::mbar_expect_tx(&g_bar, G_BYTES);
                ptx::bulk_g2s(gs, reinterpret_cast<const unsigned char *>(p.gperm) + (size_t)(z + 1) * G_BYTES, G_BYTES, &g_bar);
            }
        });
        if constexpr ((C::P - 1) & 1) __syncthreads(); // odd number of exchanges: protect buffer reuse
        // a5 + a6: trim, power, coalesced store
        float *__restrict__ out = prow + (int64_t)z * p.n_f + col0;
        if (fast) {
#pragma unroll
            for (int d = 0; d < E; ++d) {
                if (d >= 4 || d >= d0) __stcs(out + d * NT, v[d].x * v[d].x + v[d].y * v[d].y);
            }
        } else {
#pragma unroll
            for (int d = 0; d < E; ++d) {
                const int pidx = d * NT + t;
                const int64_t col = col0 + d * NT;
                if (pidx >= p.m && pidx < p.m + p.S && col < p.n_f) out[d * NT] = v[d].x * v[d].x + v[d].y * v[d].y;
            }
        }
    }
    ptx::tmem_fence_before_sync();
    __syncthreads();
    if (warp == 0) ptx::tmem_free<TC::NCOLS>(tmem_slot);
}

} // namespace fdas

// fdas.cu -- libfdas.so: kernels and C ABI of the FDAS matched-filter hot path (include/fdas.h).
//
// arXiv:1711.10855 (P:NN = PAPER.md line NN): eq.(2) P:23 evaluated by overlap-and-save with
// an on-chip FFT (eq.(3)) that is called once forward per segment and once inverse
// per matched filter ("called for every matched filter").  A CTA owns one segment at a time: the
// forward-transformed segment stays ON CHIP (tensor memory) across all n_z templates, so the spectrum
// is read from HBM once per segment and the only HBM stream of the z loop is the coalesced power-plane
// write.  The kernels are in convolve.cuh / fft_device.cuh (hot path), fft_batch.cuh (stand-alone FFT) and
// spectrum.cuh (the real-FFT + whitening step before the correlation); this file holds the C ABI.
//
// Built for sm_100a only.  No cuFFT, no CPU fallback.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>

#include "../../include/fdas.h"
#include "fft_device.cuh"
#include "convolve.cuh"
#include "fft_batch.cuh"
#include "spectrum.cuh"
#include "detect.cuh"

namespace fdas {

// -------------------------------------------------------------------------------------------
// Template preparation (off the hot path): G_z = DFT_L(pad(conj h_z)) / L in the register order of
// layout P-1 of the inverse transform, times the modulation exp(+2 pi i k NA a / Ra) that rotates
// the outputs of the first inverse pass for the shuffle exchange (fft_device.cuh).
// -------------------------------------------------------------------------------------------
template <int L>
__global__ void __launch_bounds__(Cfg<L>::NT) fdas_template_fft_kernel(const float2 *__restrict__ h, int m,
                                                                       const float2 *__restrict__ tw,
                                                                       float4 *__restrict__ gperm)
{
    using C = Cfg<L>;
    using I = InvCfg<C>;
    constexpr int E = C::E, NT = C::NT;
    extern __shared__ float2 smem[];
    const int t = threadIdx.x;
    const int z = blockIdx.x;
    const float scale = 1.0f / (float)L;
    float2 v[E];
#pragma unroll
    for (int d = 0; d < E; ++d) {
        const int j = d * NT + t;
        float2 a = make_float2(0.f, 0.f);
        if (j < m) { a = h[(size_t)z * m + j]; a.x *= scale; a.y *= -scale; } // conj(h) / L
        v[d] = a;
    }
    forward_to_inv_layout<C>(v, smem, smem + I::BUF_ELEMS, tw, t);
#pragma unroll
    for (int i = 0; i < I::NB; ++i)
#pragma unroll
        for (int k = 1; k < I::Ra; ++k) v[i * I::Ra + k] = cmulc(v[i * I::Ra + k], __ldg(tw + inv_gmod_index<C>(t, k)));
    float4 *g = gperm + (size_t)z * (E / 2) * NT + t;
#pragma unroll
    for (int q = 0; q < E / 2; ++q) g[q * NT] = make_float4(v[2 * q].x, v[2 * q].y, v[2 * q + 1].x, v[2 * q + 1].y);
}

// -------------------------------------------------------------------------------------------
// Debug FFT: natural order in, natural order out, either direction (tests only).  The inverse
// runs the hot loop's inverse_transform and then removes the unit phase it leaves on each thread's
// outputs (irrelevant to the power plane).
// -------------------------------------------------------------------------------------------
template <int L>
__global__ void __launch_bounds__(Cfg<L>::NT) fdas_debug_fft_kernel(const float2 *__restrict__ in, float2 *__restrict__ out,
                                                                    const float2 *__restrict__ tw, int inverse)
{
    using C = Cfg<L>;
    using I = InvCfg<C>;
    constexpr int E = C::E, NT = C::NT, RL = C::R(C::P - 1), BL = E / RL;
    extern __shared__ float2 smem[];
    float2 *buf0 = smem, *buf1 = smem + I::BUF_ELEMS;
    const int t = threadIdx.x;
    const float2 *x = in + (size_t)blockIdx.x * L;
    float2 *y = out + (size_t)blockIdx.x * L;
    float2 v[E];
    if (!inverse) {
#pragma unroll
        for (int d = 0; d < E; ++d) v[d] = x[d * NT + t];
        fwd_from<C, 0>(v, buf0, buf1, tw, t);
#pragma unroll
        for (int b = 0; b < BL; ++b)
#pragma unroll
            for (int d = 0; d < RL; ++d) y[nat_freq<C>(t, b, d)] = v[b * RL + d];
    } else {
#pragma unroll
        for (int i = 0; i < I::NB; ++i)
#pragma unroll
            for (int k = 0; k < I::Ra; ++k)
                v[i * I::Ra + k] = cmulc(x[inv_freq<C>(t, i, k)], __ldg(tw + inv_gmod_index<C>(t, k)));
        float2 tw0[C::R(0)];
        tw0[0] = make_float2(1.f, 0.f);
#pragma unroll
        for (int d = 1; d < C::R(0); ++d) tw0[d] = __ldg(tw + d * t);
        const InvAddr<C> A = inv_addr<C>(t);
        TwLdg<C> tws{tw, t};
        inv_stage_a<C>(v);
        inv_stage_b<C>(v, buf0, A, tws, t & 31);
        __syncthreads();
        inv_stage_c<C>(v, buf0, buf1, A, tw0, tws);
        const float2 fix = __ldg(tw + inv_fix_index<C>(t));
#pragma unroll
        for (int d = 0; d < E; ++d) y[d * NT + t] = cmul(v[d], fix);
    }
}

} // namespace fdas

// =============================================================================================
// host side
// =============================================================================================
using namespace fdas;

constexpr int HOST_CHUNKS = 8; // at most this many pieces of the host-to-device copy in fdas_detect_blockmax_host

struct fdas_plan {
    int64_t n_f;
    int z_max, z_step, n_z, m, L, S;
    int64_t n_seg;
    int n_batch;
    float4 *d_gperm;   // n_z * L complex64
    float2 *d_tw;      // L complex64
    bool has_templates;
    int last_cuda_error;
    int last_launches;
    int device;               // CUDA device the plan lives on (every call checks it)
    int grid_max[3];          // resident CTAs of the hot kernel per output mode (registers, smem, tensor memory)
    int grid_max_sym;         // same for the +-z symmetric power kernel (0: this segment length has none)
    bool sym_requested;       // fdas_plan_set_symmetry
    bool sym_detected;        // the current bank satisfies h_{-z} = conj(h_{+z}) bit for bit
    unsigned int *d_work;     // [WORK_SLOTS][2] work counters of the persistent kernel, zero between launches
    unsigned int work_seq;    // launches so far: selects the counter pair
#ifdef FDAS_EXPERIMENTS
    bool exp_nobulk;          // FDAS_EXP_NOBULK was set when the plan was created
#endif
    // buffers of fdas_convolve_host
    void *d_host_spec;
    float *d_host_power;
    void *d_host_det;
    size_t host_spec_bytes, host_power_bytes, host_det_bytes;
    void *d_cand_scratch;                     // fdas_detect_candidates: block maxima, argmaxima, row offsets
    size_t cand_scratch_bytes;
    cudaStream_t copy_stream;                 // fdas_detect_blockmax_host: chunked upload overlapping the kernel
    cudaEvent_t copy_event[HOST_CHUNKS + 1];
};

namespace {

bool supported_L(int L) { return L == 512 || L == 1024 || L == 2048 || L == 4096 || L == 8192; }

// A plan lives on the device that was current at fdas_plan_create; every later call must be made
// with that device current (its buffers, its opted-in kernel attributes).
bool on_plan_device(const fdas_plan *p)
{
    int dev = -1;
    return cudaGetDevice(&dev) == cudaSuccess && dev == p->device;
}

fdas_status cuda_fail(fdas_plan *p, cudaError_t e)
{
    if (p) p->last_cuda_error = (int)e;
    (void)cudaGetLastError();
    return FDAS_ERR_CUDA;
}

// w_L^j = exp(-i 2 pi j / L), computed in double, rounded once (eq.(3), "twiddle factors")
cudaError_t upload_twiddles(int L, float2 **d_tw)
{
    float2 *h = (float2 *)malloc(sizeof(float2) * (size_t)L);
    if (!h) return cudaErrorMemoryAllocation;
    for (int j = 0; j < L; ++j) {
        // exact octant symmetry is not needed at the tolerance; plain double evaluation
        const double a = -2.0 * M_PI * (double)j / (double)L;
        h[j].x = (float)cos(a);
        h[j].y = (float)sin(a);
    }
    cudaError_t e = cudaMalloc((void **)d_tw, sizeof(float2) * (size_t)L);
    if (e == cudaSuccess) e = cudaMemcpy(*d_tw, h, sizeof(float2) * (size_t)L, cudaMemcpyHostToDevice);
    free(h);
    return e;
}

template <int L> size_t smem_bytes() { return 2 * sizeof(float2) * (size_t)InvCfg<Cfg<L>>::BUF_ELEMS; }

// Counter pairs of the persistent kernel.  Launches take them round robin, so launches of one plan
// that run concurrently (several streams) use different pairs; a pair is re-armed by its own launch.
constexpr unsigned WORK_SLOTS = 1024;

template <int L, int OUT, bool SYM = false> cudaError_t launch_convolve(const ConvParams &cp, int grid_max, cudaStream_t st)
{
    auto kern = fdas_convolve_kernel<L, OUT, SYM>;
    constexpr size_t smem = conv_smem_bytes<Cfg<L>>();
    if (cp.n_work > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    const int64_t n_mine = cp.n_work - cp.w_begin;
    if (n_mine <= 0) return cudaSuccess;
    const unsigned grid = (unsigned)(n_mine < grid_max ? n_mine : grid_max);
    kern<<<grid, Cfg<L>::NT, smem, st>>>(cp);
    return cudaGetLastError();
}

// Once per plan, at creation: opt the hot kernel of this segment length in to its dynamic shared
// memory and size the persistent grid = resident CTAs per SM x SMs.  Resident CTAs are counted here
// from the kernel's registers and shared memory, the SM's thread / block limits and the tensor memory
// (512 columns per SM); the occupancy API reports one CTA per SM for a kernel that allocates tensor memory.
template <int L, int OUT, bool SYM = false> cudaError_t prepare_convolve(int device, int *grid_max)
{
    auto kern = fdas_convolve_kernel<L, OUT, SYM>;
    constexpr size_t smem = conv_smem_bytes<Cfg<L>>();
    constexpr int NT = Cfg<L>::NT;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    cudaFuncAttributes fa;
    e = cudaFuncGetAttributes(&fa, kern);
    if (e != cudaSuccess) return e;
    int n_sm = 0, regs_sm = 0, smem_sm = 0, smem_rsv = 0, thr_sm = 0, blk_sm = 0;
    const cudaDeviceAttr attr[6] = {cudaDevAttrMultiProcessorCount, cudaDevAttrMaxRegistersPerMultiprocessor,
                                    cudaDevAttrMaxSharedMemoryPerMultiprocessor, cudaDevAttrReservedSharedMemoryPerBlock,
                                    cudaDevAttrMaxThreadsPerMultiProcessor, cudaDevAttrMaxBlocksPerMultiprocessor};
    int *dst[6] = {&n_sm, &regs_sm, &smem_sm, &smem_rsv, &thr_sm, &blk_sm};
    for (int i = 0; i < 6; ++i) {
        e = cudaDeviceGetAttribute(dst[i], attr[i], device);
        if (e != cudaSuccess) return e;
    }
    const int regs_cta = ((fa.numRegs + 7) / 8 * 8) * NT;       // registers are allocated per warp in units of 256
    const int smem_cta = (int)smem + (int)fa.sharedSizeBytes + smem_rsv;
    int per_sm = regs_sm / regs_cta;
    if (per_sm > smem_sm / smem_cta) per_sm = smem_sm / smem_cta;
    if (per_sm > thr_sm / NT) per_sm = thr_sm / NT;
    if (per_sm > blk_sm) per_sm = blk_sm;
    if (per_sm > 512 / TmemCfg<Cfg<L>>::NCOLS) per_sm = 512 / TmemCfg<Cfg<L>>::NCOLS;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    *grid_max = per_sm * n_sm;
#ifdef FDAS_EXPERIMENTS
    // experiment knob (profiles/r2_c3_k6.md, r2_all_configs.md: grid-size sweeps); compiled out of the shipped library
    // (build.py never defines FDAS_EXPERIMENTS).  Read once per plan, at creation; values outside 1 .. resident CTAs
    // are ignored: 0 would launch an empty grid, more CTAs than fit would break the persistent kernel's one-wave rule.
    if (const char *g = getenv("FDAS_EXP_GRID")) {
        const long v = strtol(g, nullptr, 10);
        if (v >= 1 && v <= (long)*grid_max) *grid_max = (int)v;
    }
#endif
    return cudaSuccess;
}

template <int L> cudaError_t launch_template_fft(const float2 *d_h, int m, int n_z, const float2 *d_tw, float4 *d_g)
{
    auto kern = fdas_template_fft_kernel<L>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes<L>());
    if (e != cudaSuccess) return e;
    kern<<<n_z, Cfg<L>::NT, smem_bytes<L>()>>>(d_h, m, d_tw, d_g);
    return cudaGetLastError();
}

template <int L> cudaError_t launch_debug_fft(int64_t n_seg, const float2 *in, float2 *out, const float2 *d_tw, int inverse)
{
    auto kern = fdas_debug_fft_kernel<L>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes<L>());
    if (e != cudaSuccess) return e;
    kern<<<(unsigned)n_seg, Cfg<L>::NT, smem_bytes<L>()>>>(in, out, d_tw, inverse);
    return cudaGetLastError();
}

#define FDAS_DISPATCH_L(L, EXPR)                  \
    switch (L) {                                  \
    case 512: { constexpr int LL = 512; EXPR; } break;   \
    case 1024: { constexpr int LL = 1024; EXPR; } break; \
    case 2048: { constexpr int LL = 2048; EXPR; } break; \
    case 4096: { constexpr int LL = 4096; EXPR; } break; \
    case 8192: { constexpr int LL = 8192; EXPR; } break; \
    default: break;                               \
    }

} // namespace

// Host evaluation of the index maps the kernels use (fft_device.cuh): for tests without a GPU.
template <int L> static int64_t layout_query(int what, int t, int a, int b)
{
    using C = Cfg<L>;
    using I = InvCfg<C>;
    if (t < 0 || t >= C::NT) return -1;
    const InvAddr<C> A = inv_addr<C>(t);
    switch (what) {
    case FDAS_LAYOUT_GEOMETRY:
        switch (a) {
        case 0: return C::P;
        case 1: return C::E;
        case 2: return C::NT;
        case 3: return I::Ra;
        case 4: return I::Rb;
        case 5: return I::Gs;
        case 6: return I::NA;
        case 7: return I::NB;
        case 8: return I::BUF_ELEMS;
        case 9: return C::R(0);
        case 10: return C::R(1);
        default: return -1;
        }
    case FDAS_LAYOUT_FREQ: return inv_freq<C>(t, a, b);
    case FDAS_LAYOUT_GMOD: return inv_gmod_index<C>(t, a);
    case FDAS_LAYOUT_TWA: return inv_twa_index<C>(t, a, b);
    case FDAS_LAYOUT_FIX: return inv_fix_index<C>(t);
    case FDAS_LAYOUT_SHFL_SRC: return I::shfl_src_reg(a, b / I::NA, b % I::NA);
    case FDAS_LAYOUT_SHFL_DST: return I::shfl_dst_reg(a, b / I::NA, b % I::NA);
    case FDAS_LAYOUT_WRITE_A: return A.wa + I::wa_off(a, b);
    case FDAS_LAYOUT_READ_A: return A.ra + I::ra_off(a, b);
    case FDAS_LAYOUT_WRITE_B: return C::P == 4 ? A.wb + I::wb_off(a, b) : -1;
    case FDAS_LAYOUT_READ_B: return C::P == 4 ? A.rb + I::rb_off(a) : -1;
    case FDAS_LAYOUT_TW_MID: return C::P == 4 ? a * ((t % C::Lo(1)) * (C::L / (C::R(1) * C::Lo(1)))) : -1;
    default: return -1;
    }
}

// -------------------------------------------------------------------------------------------
// FP32 peak probe (measurement support, not on any path): every thread runs independent chains of dependent
// FFMA (scalar, or packed FFMA2), ITER x CHAINS per thread; bench.py --mode peak divides the flops by the
// event time.  This is what the "alu" roofline's 148 x 128 lanes x 2 x clock is checked against.
// -------------------------------------------------------------------------------------------
namespace fdas {
template <bool PACKED> __global__ void __launch_bounds__(512) fdas_alu_peak_kernel(float *out, float c, int iters)
{
    constexpr int CH = 16;
    float2 a[CH];
#pragma unroll
    for (int i = 0; i < CH; ++i) a[i] = make_float2(threadIdx.x + i, i);
    const float2 cc = make_float2(c, c);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < CH; ++i) {
            if (PACKED) a[i] = __ffma2_rn(a[(i + 1) % CH], cc, a[i]);
            else { a[i].x = fmaf(a[(i + 1) % CH].x, c, a[i].x); a[i].y = fmaf(a[(i + 1) % CH].y, c, a[i].y); }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < CH; ++i) s += a[i].x + a[i].y;
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
} // namespace fdas

// -------------------------------------------------------------------------------------------
// stand-alone batched FFT (NEXT-4; Table 1)
// -------------------------------------------------------------------------------------------
struct fdas_fft_plan {
    int n, e, device, grid_max;
    float2 *d_tw;
    // fdas_fft_exec_many: the last protocol (argument set) as an instantiated CUDA graph, and the stream it was captured on
    cudaGraphExec_t many_exec;
    cudaStream_t many_stream;
    cudaStream_t many_side[3];   // capture-time side branches (MANY_BRANCHES - 1)
    cudaEvent_t many_fork, many_join[3];
    int many_launches, many_inverse;
    int64_t many_n_fft;
    const void *many_in;
    void *many_out;
};

template <class C> static cudaError_t fft_batch_prepare(int device, int *grid_max)
{
    auto kern = fdas_fft_batch_kernel<C>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_batch_smem_bytes<C>());
    if (e != cudaSuccess) return e;
    int per_sm = 0, n_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, C::NT, fft_batch_smem_bytes<C>());
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    *grid_max = per_sm * n_sm;
    return cudaSuccess;
}
template <class C> static cudaError_t fft_batch_launch(const fdas_fft_plan *p, int64_t n_fft, const float2 *in, float2 *out,
                                                       int inverse, cudaStream_t st)
{
    const unsigned grid = (unsigned)(n_fft < p->grid_max ? n_fft : p->grid_max);
    fdas_fft_batch_kernel<C><<<grid, C::NT, fft_batch_smem_bytes<C>(), st>>>(in, out, p->d_tw, (long long)n_fft, inverse);
    return cudaGetLastError();
}
// (n, elements per thread) -> kernel configuration
#define FDAS_DISPATCH_FFT(N, E, EXPR)                                              \
    if ((N) == 512 && (E) == 8) { using CC = Cfg<512>; EXPR; }                     \
    else if ((N) == 1024 && (E) == 8) { using CC = Cfg1024E8; EXPR; }              \
    else if ((N) == 1024 && (E) == 16) { using CC = Cfg<1024>; EXPR; }             \
    else if ((N) == 2048 && (E) == 16) { using CC = Cfg<2048>; EXPR; }             \
    else if ((N) == 4096 && (E) == 16) { using CC = Cfg<4096>; EXPR; }             \
    else if ((N) == 8192 && (E) == 16) { using CC = Cfg<8192>; EXPR; }

// -------------------------------------------------------------------------------------------
// spectrum of the observation (NEXT-3): real series -> whitened complex spectrum
// -------------------------------------------------------------------------------------------
struct fdas_spectrum_plan {
    int64_t n_t, N, blk;
    int N1, N2, device;
    fdas_fft_plan *f1, *f2;   // batched transforms of length N1 and N2
    float2 *d_a, *d_b;        // scratch, N complex each
};

extern "C" {

fdas_status fdas_plan_create(fdas_plan **out, int64_t n_f, int z_max, int z_step, int template_width, int segment_len)
{
    if (!out) return FDAS_ERR_INVALID_ARG;
    if (n_f < 1 || z_max < 0 || z_step < 1 || (z_max % z_step) != 0) return FDAS_ERR_INVALID_ARG;
    if (template_width < 2 || (template_width & 1)) return FDAS_ERR_INVALID_ARG;
    if (segment_len < 2 || (segment_len & (segment_len - 1))) return FDAS_ERR_INVALID_ARG;
    if (!supported_L(segment_len)) return FDAS_ERR_UNSUPPORTED;
    if (template_width > segment_len / 2) return FDAS_ERR_INVALID_ARG;
    fdas_plan *p = (fdas_plan *)calloc(1, sizeof(fdas_plan));
    if (!p) return FDAS_ERR_ALLOC;
    p->n_f = n_f;
    p->z_max = z_max;
    p->z_step = z_step;
    p->n_z = 2 * z_max / z_step + 1;
    p->m = template_width;
    p->L = segment_len;
    p->S = segment_len - template_width;
    p->n_seg = (n_f + p->S - 1) / p->S;
    p->n_batch = 1;
#ifdef FDAS_EXPERIMENTS
    p->exp_nobulk = getenv("FDAS_EXP_NOBULK") != nullptr;
#endif
    cudaError_t e = cudaGetDevice(&p->device);
    if (e == cudaSuccess) e = cudaMalloc((void **)&p->d_gperm, sizeof(float2) * (size_t)p->n_z * (size_t)p->L);
    if (e == cudaSuccess) e = upload_twiddles(p->L, &p->d_tw);
    if (e == cudaSuccess) e = cudaMalloc((void **)&p->d_work, sizeof(unsigned int) * 2 * WORK_SLOTS);
    if (e == cudaSuccess) e = cudaMemset(p->d_work, 0, sizeof(unsigned int) * 2 * WORK_SLOTS);
    if (e == cudaSuccess) {
        const int L = p->L;
        FDAS_DISPATCH_L(L, (e = prepare_convolve<LL, OUT_POWER>(p->device, &p->grid_max[OUT_POWER])));
        if (e == cudaSuccess) { FDAS_DISPATCH_L(L, (e = prepare_convolve<LL, OUT_AMP>(p->device, &p->grid_max[OUT_AMP]))); }
        if (e == cudaSuccess) { FDAS_DISPATCH_L(L, (e = prepare_convolve<LL, OUT_BLOCKMAX>(p->device, &p->grid_max[OUT_BLOCKMAX]))); }
        // the symmetric kernel needs a free 32-column block of tensor memory: the three-pass, >= 128-thread plans
        if (e == cudaSuccess && L == 2048) e = prepare_convolve<2048, OUT_POWER, true>(p->device, &p->grid_max_sym);
        if (e == cudaSuccess && L == 4096) e = prepare_convolve<4096, OUT_POWER, true>(p->device, &p->grid_max_sym);
    }
    if (e != cudaSuccess) {
        fdas_status s = (e == cudaErrorMemoryAllocation) ? FDAS_ERR_ALLOC : FDAS_ERR_CUDA;
        (void)cudaGetLastError();
        if (p->d_gperm) cudaFree(p->d_gperm);
        if (p->d_tw) cudaFree(p->d_tw);
        if (p->d_work) cudaFree(p->d_work);
        free(p);
        return s;
    }
    *out = p;
    return FDAS_OK;
}

fdas_status fdas_plan_set_batch(fdas_plan *p, int n_batch)
{
    if (!p || n_batch < 1) return FDAS_ERR_INVALID_ARG;
    p->n_batch = n_batch;
    return FDAS_OK;
}

fdas_status fdas_set_templates(fdas_plan *p, const float *h_templates)
{
    if (!p || !h_templates) return FDAS_ERR_INVALID_ARG;
    if (!on_plan_device(p)) return FDAS_ERR_INVALID_ARG;
    const size_t bytes = sizeof(float2) * (size_t)p->n_z * (size_t)p->m;
    float2 *d_h = nullptr;
    // the bank is replaced in place: wait for every fdas_convolve still reading the old one (any stream)
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) return cuda_fail(p, e);
    e = cudaMalloc((void **)&d_h, bytes);
    if (e != cudaSuccess) { (void)cudaGetLastError(); p->last_cuda_error = (int)e; return FDAS_ERR_ALLOC; }
    e = cudaMemcpy(d_h, h_templates, bytes, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        const int L = p->L;
        FDAS_DISPATCH_L(L, e = launch_template_fft<LL>(d_h, p->m, p->n_z, p->d_tw, p->d_gperm));
    }
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    cudaFree(d_h);
    if (e != cudaSuccess) return cuda_fail(p, e);
    p->has_templates = true;
    // FDAS symmetry of the bank (SURVEY.md 8(c) note S): row n_z-1-i is the element-wise conjugate of row i, bit for
    // bit (which makes the middle row, z = 0, real).  Anything else takes the general path.
    bool sym = (p->n_z & 1) != 0;
    for (int i = 0; sym && i <= p->n_z / 2; ++i) {
        const float *a = h_templates + (size_t)2 * p->m * i, *b = h_templates + (size_t)2 * p->m * (p->n_z - 1 - i);
        for (int j = 0; j < p->m; ++j)
            if (a[2 * j] != b[2 * j] || a[2 * j + 1] != -b[2 * j + 1]) { sym = false; break; }
    }
    p->sym_detected = sym;
    return FDAS_OK;
}

fdas_status fdas_plan_set_symmetry(fdas_plan *p, int enable)
{
    if (!p) return FDAS_ERR_INVALID_ARG;
    p->sym_requested = enable != 0;
    return FDAS_OK;
}

int fdas_plan_symmetry_active(const fdas_plan *p)
{
    return p && p->sym_requested && p->sym_detected && p->grid_max_sym > 0;
}

// common part of the three entry points that enqueue the hot kernel
static fdas_status enqueue(fdas_plan *p, int out_mode, const void *d_spectrum, float *d_power, float2 *d_amp,
                           float *d_max, int *d_arg, void *cuda_stream, int64_t w_begin = 0, int64_t w_end = -1)
{
    if (!on_plan_device(p)) return FDAS_ERR_INVALID_ARG;
    if (!p->has_templates) return FDAS_ERR_NO_TEMPLATES;
    ConvParams cp;
    cp.spectrum = (const float2 *)d_spectrum;
    cp.power = d_power;
    cp.amp = d_amp;
    cp.bmax = d_max;
    cp.barg = d_arg;
    cp.gperm = p->d_gperm;
    cp.tw = p->d_tw;
    // fetch-and-add: launches on one plan may come from several host threads (one stream each), and two of them must
    // never be handed the same counter pair
    cp.work = p->d_work + 2 * (__atomic_fetch_add(&p->work_seq, 1u, __ATOMIC_RELAXED) % WORK_SLOTS);
    cp.n_f = p->n_f;
    cp.n_seg = p->n_seg;
    cp.n_work = w_end >= 0 ? w_end : p->n_seg * (int64_t)p->n_batch;
    cp.w_begin = w_begin;
    cp.n_z = p->n_z;
    cp.m = p->m;
    cp.S = p->S;
    cp.bulk_ok = ((uintptr_t)d_spectrum & 15u) == 0;
#ifdef FDAS_EXPERIMENTS
    if (p->exp_nobulk) cp.bulk_ok = 0; // experiment knob (read at plan creation): guarded loads for every segment
#endif
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaErrorInvalidValue;
    const int L = p->L;
    switch (out_mode) {
    case OUT_POWER:
        if (p->sym_requested && p->sym_detected && p->grid_max_sym > 0) {
            if (L == 2048) e = launch_convolve<2048, OUT_POWER, true>(cp, p->grid_max_sym, st);
            else e = launch_convolve<4096, OUT_POWER, true>(cp, p->grid_max_sym, st);
        } else {
            FDAS_DISPATCH_L(L, (e = launch_convolve<LL, OUT_POWER>(cp, p->grid_max[OUT_POWER], st)));
        }
        break;
    case OUT_AMP: FDAS_DISPATCH_L(L, (e = launch_convolve<LL, OUT_AMP>(cp, p->grid_max[OUT_AMP], st))); break;
    case OUT_BLOCKMAX: FDAS_DISPATCH_L(L, (e = launch_convolve<LL, OUT_BLOCKMAX>(cp, p->grid_max[OUT_BLOCKMAX], st))); break;
    default: break;
    }
    p->last_launches = 1;
    if (e != cudaSuccess) return cuda_fail(p, e);
    return FDAS_OK;
}

fdas_status fdas_convolve(fdas_plan *p, const void *d_spectrum, float *d_power, void *cuda_stream)
{
    if (!p || !d_spectrum || !d_power) return FDAS_ERR_INVALID_ARG;
    if (((uintptr_t)d_spectrum & 7u) || ((uintptr_t)d_power & 3u)) return FDAS_ERR_INVALID_ARG;
    return enqueue(p, OUT_POWER, d_spectrum, d_power, nullptr, nullptr, nullptr, cuda_stream);
}

fdas_status fdas_convolve_complex(fdas_plan *p, const void *d_spectrum, void *d_amp, void *cuda_stream)
{
    if (!p || !d_spectrum || !d_amp) return FDAS_ERR_INVALID_ARG;
    if (((uintptr_t)d_spectrum & 7u) || ((uintptr_t)d_amp & 7u)) return FDAS_ERR_INVALID_ARG;
    return enqueue(p, OUT_AMP, d_spectrum, nullptr, (float2 *)d_amp, nullptr, nullptr, cuda_stream);
}

fdas_status fdas_detect_blockmax(fdas_plan *p, const void *d_spectrum, float *d_max, int32_t *d_arg, void *cuda_stream)
{
    if (!p || !d_spectrum || !d_max || !d_arg) return FDAS_ERR_INVALID_ARG;
    if (((uintptr_t)d_spectrum & 7u) || ((uintptr_t)d_max & 3u) || ((uintptr_t)d_arg & 3u)) return FDAS_ERR_INVALID_ARG;
    return enqueue(p, OUT_BLOCKMAX, d_spectrum, nullptr, nullptr, d_max, (int *)d_arg, cuda_stream);
}

// plan-owned staging buffers of the *_host entry points: grown on demand, kept until destroy
static cudaError_t stage_reserve(void **buf, size_t *have, size_t need)
{
    if (*have >= need) return cudaSuccess;
    if (*buf) cudaFree(*buf);
    *buf = nullptr;
    *have = 0;
    cudaError_t e = cudaMalloc(buf, need);
    if (e == cudaSuccess) *have = need;
    return e;
}

// A *_host call that fails after it has enqueued something: kernels may still be queued on the caller's stream and
// copies from / into the caller's HOST buffers on the plan's copy stream.  The caller is entitled to free those buffers
// as soon as the error comes back, so wait for both streams first (their own status no longer matters).
static void host_drain(fdas_plan *p, cudaStream_t st)
{
    if (p->copy_stream) (void)cudaStreamSynchronize(p->copy_stream);
    (void)cudaStreamSynchronize(st);
    (void)cudaGetLastError();
}

// the plan's copy stream and events of the *_host entry points, created on first use
static cudaError_t ensure_copy_stream(fdas_plan *p)
{
    if (p->copy_stream) return cudaSuccess;
    cudaError_t e = cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking);
    for (int i = 0; e == cudaSuccess && i <= HOST_CHUNKS; ++i) e = cudaEventCreateWithFlags(&p->copy_event[i], cudaEventDisableTiming);
    return e;
}

fdas_status fdas_convolve_host(fdas_plan *p, const void *h_spectrum, float *h_power, void *cuda_stream)
{
    if (!p || !h_spectrum || !h_power) return FDAS_ERR_INVALID_ARG;
    if (!on_plan_device(p)) return FDAS_ERR_INVALID_ARG;
    if (!p->has_templates) return FDAS_ERR_NO_TEMPLATES;
    const size_t sb = sizeof(float2) * (size_t)p->n_batch * (size_t)p->n_f;
    const size_t pb = sizeof(float) * (size_t)p->n_batch * (size_t)p->n_z * (size_t)p->n_f;
    cudaError_t e = stage_reserve(&p->d_host_spec, &p->host_spec_bytes, sb);
    if (e == cudaSuccess) e = stage_reserve((void **)&p->d_host_power, &p->host_power_bytes, pb);
    if (e != cudaSuccess) { (void)cudaGetLastError(); p->last_cuda_error = (int)e; return FDAS_ERR_ALLOC; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    e = cudaMemcpyAsync(p->d_host_spec, h_spectrum, sb, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(p, e);
    // From here on work is in flight: every error return drains it first (host_drain).
    // The plane is 100 x the spectrum: its way back dominates.  The work items are launched in up to HOST_CHUNKS
    // pieces of at least a wave each, and every piece's columns start their way back (2-D copies on the plan's copy
    // stream) while the next piece is computed.
    const int64_t n_work = p->n_seg * (int64_t)p->n_batch;
    const int64_t waves = (n_work + p->grid_max[OUT_POWER] - 1) / p->grid_max[OUT_POWER];
    const int n_chunks = (int)(waves > HOST_CHUNKS ? HOST_CHUNKS : waves);
    if (n_chunks <= 1) {
        fdas_status s = fdas_convolve(p, p->d_host_spec, p->d_host_power, cuda_stream);
        if (s != FDAS_OK) { host_drain(p, st); return s; }
        e = cudaMemcpyAsync(h_power, p->d_host_power, pb, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { host_drain(p, st); return cuda_fail(p, e); }
        return FDAS_OK;
    }
    e = ensure_copy_stream(p);
    if (e != cudaSuccess) { host_drain(p, st); return cuda_fail(p, e); }
    const size_t pitch = sizeof(float) * (size_t)p->n_f;
    for (int c = 0; c < n_chunks; ++c) {
        const int64_t w0 = n_work * c / n_chunks, w1 = n_work * (c + 1) / n_chunks;
        fdas_status s = enqueue(p, OUT_POWER, p->d_host_spec, p->d_host_power, nullptr, nullptr, nullptr, cuda_stream, w0, w1);
        if (s != FDAS_OK) { host_drain(p, st); return s; }
        e = cudaEventRecord(p->copy_event[c], st);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(p->copy_stream, p->copy_event[c], 0);
        for (int64_t bi = w0 / p->n_seg; e == cudaSuccess && bi <= (w1 - 1) / p->n_seg; ++bi) { // batch items the piece touches
            const int64_t sa = bi == w0 / p->n_seg ? w0 % p->n_seg : 0;
            const int64_t sz = bi == (w1 - 1) / p->n_seg ? (w1 - 1) % p->n_seg + 1 : p->n_seg;
            const int64_t c0 = sa * p->S, c1 = sz * p->S < p->n_f ? sz * p->S : p->n_f;
            const size_t off = (size_t)bi * (size_t)p->n_z * (size_t)p->n_f + (size_t)c0;
            e = cudaMemcpy2DAsync(h_power + off, pitch, p->d_host_power + off, pitch, sizeof(float) * (size_t)(c1 - c0), (size_t)p->n_z,
                                  cudaMemcpyDeviceToHost, p->copy_stream);
        }
        if (e != cudaSuccess) { host_drain(p, st); return cuda_fail(p, e); }
    }
    p->last_launches = n_chunks;
    e = cudaEventRecord(p->copy_event[HOST_CHUNKS], p->copy_stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(st, p->copy_event[HOST_CHUNKS], 0);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { host_drain(p, st); return cuda_fail(p, e); }
    return FDAS_OK;
}

// Spectrum from HOST memory -> block maxima in DEVICE arrays d_max / d_arg, enqueued on the caller's stream (nothing
// is downloaded, nothing synchronised): the common front of fdas_detect_blockmax_host and fdas_detect_candidates_host.
// On an error it has drained what it had enqueued.
static fdas_status blockmax_from_host(fdas_plan *p, const void *h_spectrum, float *d_max, int32_t *d_arg, void *cuda_stream)
{
    const size_t sb = sizeof(float2) * (size_t)p->n_batch * (size_t)p->n_f;
    cudaError_t e = stage_reserve(&p->d_host_spec, &p->host_spec_bytes, sb);
    if (e != cudaSuccess) { (void)cudaGetLastError(); p->last_cuda_error = (int)e; return FDAS_ERR_ALLOC; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // The spectrum goes up in HOST_CHUNKS pieces on a plan-owned copy stream and every piece's segments are launched
    // as soon as it has arrived, so that all but the first piece of the host-to-device copy hides behind the kernel.
    // The pieces are ranges of work items = (batch item, segment) in order, i.e. contiguous ranges of the input.
    const int64_t n_work = p->n_seg * (int64_t)p->n_batch;
    // Every piece is about one full wave of the persistent grid or more: smaller launches would leave SMs idle.
    // A call that is a single wave anyway goes the plain way: copy and launch on the caller's stream.
    const int64_t waves = (n_work + p->grid_max[OUT_BLOCKMAX] - 1) / p->grid_max[OUT_BLOCKMAX];
    const int n_chunks = (int)(waves > HOST_CHUNKS ? HOST_CHUNKS : waves);
    if (n_chunks <= 1) {
        e = cudaMemcpyAsync(p->d_host_spec, h_spectrum, sb, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return cuda_fail(p, e);
        fdas_status s1 = fdas_detect_blockmax(p, p->d_host_spec, d_max, d_arg, cuda_stream);
        if (s1 != FDAS_OK) { host_drain(p, st); return s1; }
        return FDAS_OK;
    }
    e = ensure_copy_stream(p);
    if (e != cudaSuccess) return cuda_fail(p, e);
    e = cudaEventRecord(p->copy_event[HOST_CHUNKS], st);                  // the copies start after the caller's earlier work
    if (e == cudaSuccess) e = cudaStreamWaitEvent(p->copy_stream, p->copy_event[HOST_CHUNKS], 0);
    if (e != cudaSuccess) { host_drain(p, st); return cuda_fail(p, e); }
    size_t copied = 0; // complex elements of the flattened [n_batch][n_f] spectrum on the device so far
    for (int c = 0; c < n_chunks; ++c) {
        const int64_t w0 = n_work * c / n_chunks, w1 = n_work * (c + 1) / n_chunks;
        // the last item of the piece is (bi, seg) = ((w1-1) / n_seg, (w1-1) % n_seg): it reads bins up to seg*S - m/2 + L
        const int64_t bi = (w1 - 1) / p->n_seg, seg = (w1 - 1) % p->n_seg;
        int64_t hi = seg * (int64_t)p->S - p->m / 2 + p->L;
        if (hi > p->n_f) hi = p->n_f;
        size_t upto = (size_t)bi * (size_t)p->n_f + (size_t)hi;
        if (c == n_chunks - 1) upto = (size_t)p->n_batch * (size_t)p->n_f;
        if (upto > copied) {
            e = cudaMemcpyAsync((float2 *)p->d_host_spec + copied, (const float2 *)h_spectrum + copied, sizeof(float2) * (upto - copied),
                                cudaMemcpyHostToDevice, p->copy_stream);
            copied = upto;
        }
        if (e == cudaSuccess) e = cudaEventRecord(p->copy_event[c], p->copy_stream);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(st, p->copy_event[c], 0);
        if (e != cudaSuccess) { host_drain(p, st); return cuda_fail(p, e); }
        fdas_status s = enqueue(p, OUT_BLOCKMAX, p->d_host_spec, nullptr, nullptr, d_max, (int *)d_arg, cuda_stream, w0, w1);
        if (s != FDAS_OK) { host_drain(p, st); return s; }
    }
    p->last_launches = n_chunks;
    return FDAS_OK;
}

fdas_status fdas_detect_blockmax_host(fdas_plan *p, const void *h_spectrum, float *h_max, int32_t *h_arg, void *cuda_stream)
{
    if (!p || !h_spectrum || !h_max || !h_arg) return FDAS_ERR_INVALID_ARG;
    if (!on_plan_device(p)) return FDAS_ERR_INVALID_ARG;
    if (!p->has_templates) return FDAS_ERR_NO_TEMPLATES;
    const size_t nb = (size_t)p->n_batch * (size_t)p->n_z * (size_t)p->n_seg; // entries of each result array
    cudaError_t e = stage_reserve(&p->d_host_det, &p->host_det_bytes, 8 * nb);
    if (e != cudaSuccess) { (void)cudaGetLastError(); p->last_cuda_error = (int)e; return FDAS_ERR_ALLOC; }
    float *d_max = (float *)p->d_host_det;
    int32_t *d_arg = (int32_t *)p->d_host_det + nb;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    fdas_status s = blockmax_from_host(p, h_spectrum, d_max, d_arg, cuda_stream);
    if (s != FDAS_OK) return s;
    e = cudaMemcpyAsync(h_max, d_max, 4 * nb, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h_arg, d_arg, 4 * nb, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { host_drain(p, st); return cuda_fail(p, e); }
    return FDAS_OK;
}

// The plan-owned scratch of fdas_detect_candidates[_host]: [nb] float maxima | [nb] int32 offsets | [n_rows + 1] int32.
struct CandScratch { float *d_max; int32_t *d_arg; int *d_rows; size_t nb; int n_rows; };

static fdas_status cand_scratch(fdas_plan *p, int capacity, CandScratch *cs)
{
    const size_t nb = (size_t)p->n_batch * (size_t)p->n_z * (size_t)p->n_seg;
    if (capacity < 0 || nb >= ((size_t)1 << 31)) return FDAS_ERR_INVALID_ARG;
    const int n_rows = p->n_batch * p->n_z;
    cudaError_t e = stage_reserve(&p->d_cand_scratch, &p->cand_scratch_bytes, 8 * nb + 4 * ((size_t)n_rows + 1));
    if (e != cudaSuccess) { (void)cudaGetLastError(); p->last_cuda_error = (int)e; return FDAS_ERR_ALLOC; }
    cs->d_max = (float *)p->d_cand_scratch;
    cs->d_arg = (int32_t *)p->d_cand_scratch + nb;
    cs->d_rows = (int *)p->d_cand_scratch + 2 * nb;
    cs->nb = nb;
    cs->n_rows = n_rows;
    return FDAS_OK;
}

// block maxima (already enqueued on st) -> candidate list and counts, three small launches on st
static cudaError_t cand_compact(fdas_plan *p, const CandScratch &cs, float threshold, int capacity, fdas_candidate *d_cand,
                                int32_t *d_count, cudaStream_t st)
{
    const unsigned row_ctas = (unsigned)((cs.n_rows + 7) / 8); // 8 warps per CTA, one warp per (item, row)
    fdas_cand_count_kernel<<<row_ctas, 256, 0, st>>>(cs.d_max, cs.n_rows, (long long)p->n_seg, threshold, cs.d_rows);
    fdas_cand_scan_kernel<<<1, 1024, 0, st>>>(cs.d_rows, cs.n_rows, capacity, d_count);
    fdas_cand_scatter_kernel<<<row_ctas, 256, 0, st>>>(cs.d_max, cs.d_arg, cs.n_rows, p->n_z, (long long)p->n_seg, p->S, threshold,
                                                       cs.d_rows, capacity, d_cand);
    p->last_launches += 3;
    return cudaGetLastError();
}

fdas_status fdas_detect_candidates(fdas_plan *p, const void *d_spectrum, float threshold, int capacity, fdas_candidate *d_cand,
                                   int32_t *d_count, void *cuda_stream)
{
    if (!p || !d_spectrum || !d_count || (!d_cand && capacity > 0)) return FDAS_ERR_INVALID_ARG;
    if (((uintptr_t)d_spectrum & 7u) || ((uintptr_t)d_cand & 3u) || ((uintptr_t)d_count & 3u)) return FDAS_ERR_INVALID_ARG;
    if (!on_plan_device(p)) return FDAS_ERR_INVALID_ARG;
    if (!p->has_templates) return FDAS_ERR_NO_TEMPLATES;
    CandScratch cs;
    fdas_status s = cand_scratch(p, capacity, &cs);
    if (s != FDAS_OK) return s;
    s = enqueue(p, OUT_BLOCKMAX, d_spectrum, nullptr, nullptr, cs.d_max, (int *)cs.d_arg, cuda_stream);
    if (s != FDAS_OK) return s;
    cudaError_t e = cand_compact(p, cs, threshold, capacity, d_cand, d_count, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(p, e);
    return FDAS_OK;
}

fdas_status fdas_detect_candidates_host(fdas_plan *p, const void *h_spectrum, float threshold, int capacity, fdas_candidate *h_cand,
                                        int32_t *h_count, void *cuda_stream)
{
    if (!p || !h_spectrum || !h_count || (!h_cand && capacity > 0)) return FDAS_ERR_INVALID_ARG;
    if (!on_plan_device(p)) return FDAS_ERR_INVALID_ARG;
    if (!p->has_templates) return FDAS_ERR_NO_TEMPLATES;
    CandScratch cs;
    fdas_status s = cand_scratch(p, capacity, &cs);
    if (s != FDAS_OK) return s;
    // the device copies of the two results: 16 * capacity + 8 bytes behind the spectrum's staging-independent buffer
    const size_t out_bytes = sizeof(fdas_candidate) * (size_t)capacity + 8;
    cudaError_t e = stage_reserve(&p->d_host_det, &p->host_det_bytes, out_bytes);
    if (e != cudaSuccess) { (void)cudaGetLastError(); p->last_cuda_error = (int)e; return FDAS_ERR_ALLOC; }
    int32_t *d_count = (int32_t *)p->d_host_det;
    fdas_candidate *d_cand = (fdas_candidate *)((unsigned char *)p->d_host_det + 8);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    s = blockmax_from_host(p, h_spectrum, cs.d_max, cs.d_arg, cuda_stream);
    if (s != FDAS_OK) return s;
    e = cand_compact(p, cs, threshold, capacity, d_cand, d_count, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h_count, d_count, 8, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && capacity > 0)
        e = cudaMemcpyAsync(h_cand, d_cand, sizeof(fdas_candidate) * (size_t)capacity, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { host_drain(p, st); return cuda_fail(p, e); }
    return FDAS_OK;
}

fdas_status fdas_plan_destroy(fdas_plan *p)
{
    if (!p) return FDAS_OK;
    if (p->d_gperm) cudaFree(p->d_gperm);
    if (p->d_tw) cudaFree(p->d_tw);
    if (p->d_work) cudaFree(p->d_work);
    if (p->d_host_spec) cudaFree(p->d_host_spec);
    if (p->d_host_power) cudaFree(p->d_host_power);
    if (p->d_host_det) cudaFree(p->d_host_det);
    if (p->d_cand_scratch) cudaFree(p->d_cand_scratch);
    if (p->copy_stream) {
        for (int i = 0; i <= HOST_CHUNKS; ++i) if (p->copy_event[i]) cudaEventDestroy(p->copy_event[i]);
        cudaStreamDestroy(p->copy_stream);
    }
    (void)cudaGetLastError();
    free(p);
    return FDAS_OK;
}

int fdas_plan_nz(const fdas_plan *p) { return p ? p->n_z : 0; }
int fdas_plan_step(const fdas_plan *p) { return p ? p->S : 0; }
int64_t fdas_plan_nseg(const fdas_plan *p) { return p ? p->n_seg : 0; }
int fdas_plan_batch(const fdas_plan *p) { return p ? p->n_batch : 0; }
int fdas_plan_grid(const fdas_plan *p) { return p ? p->grid_max[OUT_POWER] : 0; }
int fdas_plan_last_launch_count(const fdas_plan *p) { return p ? p->last_launches : 0; }
int fdas_plan_last_cuda_error(const fdas_plan *p) { return p ? p->last_cuda_error : -1; }

fdas_status fdas_fft_plan_create(fdas_fft_plan **out, int n, int elems_per_thread)
{
    if (!out) return FDAS_ERR_INVALID_ARG;
    if (!supported_L(n)) return FDAS_ERR_UNSUPPORTED;
    int e_thr = elems_per_thread ? elems_per_thread : (n == 512 ? 8 : 16);
    if (!((e_thr == 8 && (n == 512 || n == 1024)) || (e_thr == 16 && n >= 1024))) return FDAS_ERR_UNSUPPORTED;
    fdas_fft_plan *p = (fdas_fft_plan *)calloc(1, sizeof(fdas_fft_plan));
    if (!p) return FDAS_ERR_ALLOC;
    p->n = n;
    p->e = e_thr;
    cudaError_t e = cudaGetDevice(&p->device);
    if (e == cudaSuccess) e = upload_twiddles(n, &p->d_tw);
    if (e == cudaSuccess) { FDAS_DISPATCH_FFT(n, e_thr, (e = fft_batch_prepare<CC>(p->device, &p->grid_max))) }
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        if (p->d_tw) cudaFree(p->d_tw);
        free(p);
        return e == cudaErrorMemoryAllocation ? FDAS_ERR_ALLOC : FDAS_ERR_CUDA;
    }
    *out = p;
    return FDAS_OK;
}

fdas_status fdas_fft_exec(fdas_fft_plan *p, int64_t n_fft, const void *d_in, void *d_out, int inverse, void *cuda_stream)
{
    if (!p || !d_in || !d_out || n_fft < 0 || d_in == d_out) return FDAS_ERR_INVALID_ARG;
    if (((uintptr_t)d_in & 7u) || ((uintptr_t)d_out & 7u)) return FDAS_ERR_INVALID_ARG;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device) return FDAS_ERR_INVALID_ARG;
    if (n_fft == 0) return FDAS_OK;
    cudaError_t e = cudaErrorInvalidValue;
    FDAS_DISPATCH_FFT(p->n, p->e, (e = fft_batch_launch<CC>(p, n_fft, (const float2 *)d_in, (float2 *)d_out, inverse,
                                                            (cudaStream_t)cuda_stream)))
    if (e != cudaSuccess) { (void)cudaGetLastError(); return FDAS_ERR_CUDA; }
    return FDAS_OK;
}

// launch i transforms sequences [i * n_fft, (i+1) * n_fft): 1000 x 100 walks 100 000 distinct sequences through HBM
static fdas_status fft_exec_loop(fdas_fft_plan *p, int n_launches, int64_t n_fft, const void *d_in, void *d_out, int inverse,
                                 void *cuda_stream)
{
    const size_t stride = (size_t)n_fft * (size_t)p->n;   // complex64 elements per launch
    for (int i = 0; i < n_launches; ++i) {
        fdas_status s = fdas_fft_exec(p, n_fft, (const float2 *)d_in + i * stride, (float2 *)d_out + i * stride, inverse, cuda_stream);
        if (s != FDAS_OK) return s;
    }
    return FDAS_OK;
}

fdas_status fdas_fft_exec_many(fdas_fft_plan *p, int n_launches, int64_t n_fft, const void *d_in, void *d_out, int inverse,
                               void *cuda_stream)
{
    if (!p || !d_in || !d_out || n_launches < 0 || n_fft < 0 || d_in == d_out) return FDAS_ERR_INVALID_ARG;
    if (((uintptr_t)d_in & 7u) || ((uintptr_t)d_out & 7u)) return FDAS_ERR_INVALID_ARG;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device) return FDAS_ERR_INVALID_ARG;
    if (n_launches == 0 || n_fft == 0) return FDAS_OK;
    // A handful of launches go out one by one.  A long protocol is launch-rate bound that way (1000 launches cost 4.1 ms
    // of host-side launch intervals for 0.3 ms of work, profiles/r2_side_benchmarks.md), so it is recorded once as a CUDA
    // graph of the same n_launches kernels and the graph is launched; it is kept for the next call with the same
    // arguments.  The launches touch disjoint sequences, so nothing orders them but the stream they used to share: the
    // graph says so, as MANY_BRANCHES chains (launch i follows launch i - MANY_BRANCHES), which lets the GPU start a
    // launch while its neighbours run (one chain: 2.65 ms for 1000 x 100, a dependent launch every 2.6 us).
    constexpr int GRAPH_FROM = 8, MANY_BRANCHES = 4;
    if (n_launches < GRAPH_FROM) return fft_exec_loop(p, n_launches, n_fft, d_in, d_out, inverse, cuda_stream);
    inverse = inverse != 0;
    const bool hit = p->many_exec && p->many_launches == n_launches && p->many_n_fft == n_fft && p->many_in == d_in &&
                     p->many_out == d_out && p->many_inverse == inverse;
    if (!hit) {
        if (p->many_exec) { cudaGraphExecDestroy(p->many_exec); p->many_exec = nullptr; }
        cudaError_t e = cudaSuccess;
        if (!p->many_stream) {
            e = cudaStreamCreateWithFlags(&p->many_stream, cudaStreamNonBlocking);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->many_fork, cudaEventDisableTiming);
            for (int b = 0; b < MANY_BRANCHES - 1 && e == cudaSuccess; ++b) {
                e = cudaStreamCreateWithFlags(&p->many_side[b], cudaStreamNonBlocking);
                if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->many_join[b], cudaEventDisableTiming);
            }
        }
        if (e == cudaSuccess) e = cudaStreamBeginCapture(p->many_stream, cudaStreamCaptureModeThreadLocal);
        if (e != cudaSuccess) { (void)cudaGetLastError(); return FDAS_ERR_CUDA; }
        // fork the side branches off the capturing stream, deal the launches round robin, join them again
        e = cudaEventRecord(p->many_fork, p->many_stream);
        for (int b = 0; b < MANY_BRANCHES - 1 && e == cudaSuccess; ++b) e = cudaStreamWaitEvent(p->many_side[b], p->many_fork, 0);
        fdas_status s = e == cudaSuccess ? FDAS_OK : FDAS_ERR_CUDA;
        const size_t stride = (size_t)n_fft * (size_t)p->n;
        for (int i = 0; i < n_launches && s == FDAS_OK; ++i) {
            cudaStream_t bs = (i % MANY_BRANCHES) ? p->many_side[i % MANY_BRANCHES - 1] : p->many_stream;
            s = fdas_fft_exec(p, n_fft, (const float2 *)d_in + i * stride, (float2 *)d_out + i * stride, inverse, (void *)bs);
        }
        for (int b = 0; b < MANY_BRANCHES - 1 && s == FDAS_OK; ++b) {
            e = cudaEventRecord(p->many_join[b], p->many_side[b]);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(p->many_stream, p->many_join[b], 0);
            if (e != cudaSuccess) s = FDAS_ERR_CUDA;
        }
        cudaGraph_t graph = nullptr;
        e = cudaStreamEndCapture(p->many_stream, &graph);   // also ends a capture that a failed launch invalidated
        if (s == FDAS_OK && e == cudaSuccess) e = cudaGraphInstantiate(&p->many_exec, graph, 0);
        if (graph) cudaGraphDestroy(graph);
        if (s != FDAS_OK || e != cudaSuccess) {
            (void)cudaGetLastError();
            p->many_exec = nullptr;
            return s != FDAS_OK ? s : FDAS_ERR_CUDA;
        }
        p->many_launches = n_launches;
        p->many_n_fft = n_fft;
        p->many_in = d_in;
        p->many_out = d_out;
        p->many_inverse = inverse;
    }
    if (cudaGraphLaunch(p->many_exec, (cudaStream_t)cuda_stream) != cudaSuccess) { (void)cudaGetLastError(); return FDAS_ERR_CUDA; }
    return FDAS_OK;
}

fdas_status fdas_fft_plan_destroy(fdas_fft_plan *p)
{
    if (!p) return FDAS_OK;
    if (p->many_exec) cudaGraphExecDestroy(p->many_exec);
    if (p->many_stream) cudaStreamDestroy(p->many_stream);
    if (p->many_fork) cudaEventDestroy(p->many_fork);
    for (int b = 0; b < 3; ++b) {
        if (p->many_side[b]) cudaStreamDestroy(p->many_side[b]);
        if (p->many_join[b]) cudaEventDestroy(p->many_join[b]);
    }
    if (p->d_tw) cudaFree(p->d_tw);
    (void)cudaGetLastError();
    free(p);
    return FDAS_OK;
}

int fdas_fft_plan_elems_per_thread(const fdas_fft_plan *p) { return p ? p->e : 0; }
int fdas_fft_plan_grid(const fdas_fft_plan *p) { return p ? p->grid_max : 0; }

fdas_status fdas_spectrum_plan_destroy(fdas_spectrum_plan *p)
{
    if (!p) return FDAS_OK;
    fdas_fft_plan_destroy(p->f1);
    fdas_fft_plan_destroy(p->f2);
    if (p->d_a) cudaFree(p->d_a);
    if (p->d_b) cudaFree(p->d_b);
    (void)cudaGetLastError();
    free(p);
    return FDAS_OK;
}

fdas_status fdas_spectrum_plan_create(fdas_spectrum_plan **out, int64_t n_samples, int64_t whiten_block)
{
    if (!out || n_samples < 4 || (n_samples & (n_samples - 1))) return FDAS_ERR_INVALID_ARG;
    int k = 0;
    while (((int64_t)1 << k) < n_samples / 2) ++k;          // N = 2^k complex points
    if (k < 18 || k > 26) return FDAS_ERR_UNSUPPORTED;       // N = N1 N2 with both factors in 512 .. 8192
    fdas_spectrum_plan *p = (fdas_spectrum_plan *)calloc(1, sizeof(fdas_spectrum_plan));
    if (!p) return FDAS_ERR_ALLOC;
    p->n_t = n_samples;
    p->N = n_samples / 2;
    p->blk = whiten_block > 0 ? whiten_block : 0;
    p->N1 = 1 << ((k + 1) / 2);
    p->N2 = 1 << (k / 2);
    fdas_status s = fdas_fft_plan_create(&p->f1, p->N1, 0);
    if (s == FDAS_OK) s = fdas_fft_plan_create(&p->f2, p->N2, 0);
    cudaError_t e = cudaSuccess;
    if (s == FDAS_OK) e = cudaGetDevice(&p->device);
    if (s == FDAS_OK && e == cudaSuccess) e = cudaMalloc((void **)&p->d_a, sizeof(float2) * (size_t)p->N);
    if (s == FDAS_OK && e == cudaSuccess) e = cudaMalloc((void **)&p->d_b, sizeof(float2) * (size_t)p->N);
    if (s != FDAS_OK || e != cudaSuccess) {
        (void)cudaGetLastError();
        fdas_spectrum_plan_destroy(p);
        return s != FDAS_OK ? s : (e == cudaErrorMemoryAllocation ? FDAS_ERR_ALLOC : FDAS_ERR_CUDA);
    }
    *out = p;
    return FDAS_OK;
}

fdas_status fdas_spectrum_exec(fdas_spectrum_plan *p, const float *d_series, void *d_spectrum, void *cuda_stream)
{
    if (!p || !d_series || !d_spectrum) return FDAS_ERR_INVALID_ARG;
    if (((uintptr_t)d_series & 7u) || ((uintptr_t)d_spectrum & 7u)) return FDAS_ERR_INVALID_ARG;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device) return FDAS_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const float2 *z = (const float2 *)d_series;  // z[n] = x[2n] + i x[2n+1], viewed as [N1][N2]
    const dim3 thr(32, 8);
    // z [N1][N2] -> a [N2][N1];  N2 transforms of length N1: a -> b [n2][k1]
    fdas_transpose_kernel<false><<<dim3(p->N2 / 32, p->N1 / 32), thr, 0, st>>>(z, p->d_a, p->N1, p->N2, p->N);
    fdas_status s = fdas_fft_exec(p->f1, p->N2, p->d_a, p->d_b, 0, cuda_stream);
    if (s != FDAS_OK) return s;
    // b [N2][N1] times w_N^{n2 k1} -> a [k1][n2];  N1 transforms of length N2: a -> b [k1][k2] = Z[k1 + N1 k2]
    fdas_transpose_kernel<true><<<dim3(p->N1 / 32, p->N2 / 32), thr, 0, st>>>(p->d_b, p->d_a, p->N2, p->N1, p->N);
    s = fdas_fft_exec(p->f2, p->N1, p->d_a, p->d_b, 0, cuda_stream);
    if (s != FDAS_OK) return s;
    // b [N1][N2] -> a [k2][k1]: Z in natural order;  then separate the two real transforms and whiten
    fdas_transpose_kernel<false><<<dim3(p->N2 / 32, p->N1 / 32), thr, 0, st>>>(p->d_b, p->d_a, p->N1, p->N2, p->N);
    const long long width = p->blk > 0 ? p->blk : 4096;
    const long long n_cta = (p->N + width - 1) / width;
    if (n_cta > 0x7fffffffLL) return FDAS_ERR_INVALID_ARG;
    fdas_rfft_whiten_kernel<<<(unsigned)n_cta, 256, 0, st>>>(p->d_a, (float2 *)d_spectrum, p->N, p->blk);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { (void)cudaGetLastError(); return FDAS_ERR_CUDA; }
    return FDAS_OK;
}

int64_t fdas_spectrum_plan_bins(const fdas_spectrum_plan *p) { return p ? p->N : 0; }

const char *fdas_status_string(fdas_status s)
{
    switch (s) {
    case FDAS_OK: return "FDAS_OK";
    case FDAS_ERR_INVALID_ARG: return "FDAS_ERR_INVALID_ARG";
    case FDAS_ERR_UNSUPPORTED: return "FDAS_ERR_UNSUPPORTED";
    case FDAS_ERR_ALLOC: return "FDAS_ERR_ALLOC";
    case FDAS_ERR_NO_TEMPLATES: return "FDAS_ERR_NO_TEMPLATES";
    case FDAS_ERR_CUDA: return "FDAS_ERR_CUDA";
    case FDAS_ERR_TOO_LARGE: return "FDAS_ERR_TOO_LARGE";
    }
    return "FDAS_ERR_UNKNOWN";
}

fdas_status fdas_debug_fft(int segment_len, int64_t n_seg, const void *d_in, void *d_out, int inverse)
{
    if (!d_in || !d_out || n_seg < 0) return FDAS_ERR_INVALID_ARG;
    if (!supported_L(segment_len)) return FDAS_ERR_UNSUPPORTED;
    if (n_seg == 0) return FDAS_OK;
    float2 *d_tw = nullptr;
    cudaError_t e = upload_twiddles(segment_len, &d_tw);
    if (e == cudaSuccess) {
        FDAS_DISPATCH_L(segment_len, e = launch_debug_fft<LL>(n_seg, (const float2 *)d_in, (float2 *)d_out, d_tw, inverse));
    }
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (d_tw) cudaFree(d_tw);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return FDAS_ERR_CUDA; }
    return FDAS_OK;
}

fdas_status fdas_debug_alu_peak(int packed, double *tflops_out, double *ms_out)
{
    if (!tflops_out) return FDAS_ERR_INVALID_ARG;
    int dev = 0, n_sm = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    float *d_out = nullptr;
    const int blocks = 4 * (n_sm > 0 ? n_sm : 1), iters = 4000;
    if (e == cudaSuccess) e = cudaMalloc((void **)&d_out, sizeof(float) * 512 * (size_t)blocks);
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    float ms = 0.f;
    if (e == cudaSuccess) {
        for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) { // the last of three launches is the timed one
            cudaEventRecord(e0);
            if (packed) fdas_alu_peak_kernel<true><<<blocks, 512>>>(d_out, 1.0001f, iters);
            else fdas_alu_peak_kernel<false><<<blocks, 512>>>(d_out, 1.0001f, iters);
            cudaEventRecord(e1);
            e = cudaEventSynchronize(e1);
            if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        }
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (d_out) cudaFree(d_out);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return FDAS_ERR_CUDA; }
    const double flops = 2.0 * 2.0 * 16.0 * (double)iters * 512.0 * (double)blocks; // 2 flops x 2 lanes x chains x iters x threads
    *tflops_out = flops / ((double)ms * 1e-3) / 1e12;
    if (ms_out) *ms_out = ms;
    return FDAS_OK;
}

int64_t fdas_debug_layout(int segment_len, int what, int t, int a, int b)
{
    int64_t r = -1;
    FDAS_DISPATCH_L(segment_len, r = layout_query<LL>(what, t, a, b));
    return r;
}

} // extern "C"

// -------------------------------------------------------------------------------------------
// fdas_convolve_noalloc: the plan-less entry point for callers that may not allocate device memory
// (include/fdas.h says who they are).  Everything a plan would have cudaMalloc'ed -- work counters, twiddle
// table, transformed bank -- sits in ONE array that is part of the library image, so the CUDA runtime
// places a copy on every GPU that loads libfdas.so and no call here ever asks the driver for memory.
//
// The name `noalloc_scratch` means two different things.  Inside device code it is the array.  Inside host
// code it is only a handle the runtime knows the array by: handing `noalloc_scratch` itself to a kernel
// passes a HOST address (a fault on the GPU, or on machines where the GPU can read host memory a quiet
// scribble over host data).  Host code therefore asks the runtime for the device address, once per GPU
// and with that GPU current (noalloc_device below), and gives the kernels that.
// -------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char noalloc_scratch[FDAS_NOALLOC_SCRATCH_BYTES];

namespace fdas {
// Part (1) of a call: w_L^j = exp(-i 2 pi j / L) for this L (evaluated in double, rounded once, like the host
// table of a plan) and the two work counters back to zero -- whatever the previous call, or a launch
// that never finished, left in them.
__global__ void __launch_bounds__(256) fdas_noalloc_init_kernel(float2 *__restrict__ tw, int L, unsigned int *__restrict__ work)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < L) {
        double s, c;
        sincospi(-2.0 * (double)j / (double)L, &s, &c);
        tw[j] = make_float2((float)c, (float)s);
    }
    if (j == 0) { work[0] = 0u; work[1] = 0u; }
}
} // namespace fdas

namespace {

constexpr size_t NOALLOC_WORK_OFF = 0, NOALLOC_TW_OFF = 256, NOALLOC_BANK_OFF = 256 + 8 * 8192;
static_assert(NOALLOC_BANK_OFF + 8 * (size_t)FDAS_NOALLOC_MAX_BANK == FDAS_NOALLOC_SCRATCH_BYTES, "scratch layout");
constexpr int NOALLOC_MAX_DEVICES = 64;

struct NoallocDevice {
    bool ready;
    unsigned char *base; // DEVICE address of noalloc_scratch on this GPU
    int grid_max[5];     // persistent grid of the power kernel for L = 512 << i
};
NoallocDevice noalloc_dev[NOALLOC_MAX_DEVICES];
std::mutex noalloc_mutex;

int noalloc_L_index(int L) { return L == 512 ? 0 : L == 1024 ? 1 : L == 2048 ? 2 : L == 4096 ? 3 : 4; }

template <int L> cudaError_t noalloc_prepare(int dev, int *grid_max)
{
    cudaError_t e = prepare_convolve<L, OUT_POWER>(dev, grid_max);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(fdas_template_fft_kernel<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes<L>());
    return e;
}

// part (2) of a call: fdas_set_templates' kernel, but on the caller's stream and writing the scratch bank
template <int L> cudaError_t noalloc_bank(const float2 *d_h, int m, int n_z, const float2 *tw, float4 *bank, cudaStream_t st)
{
    fdas_template_fft_kernel<L><<<(unsigned)n_z, Cfg<L>::NT, smem_bytes<L>(), st>>>(d_h, m, tw, bank);
    return cudaGetLastError();
}

// First call on a GPU (that GPU is current): device address of the array, opt-in shared-memory sizes of the two
// kernels for every segment length, grid sizes.  Host-side calls only; nothing is allocated, nothing enqueued.
cudaError_t noalloc_device(int dev, const NoallocDevice **out)
{
    std::lock_guard<std::mutex> lock(noalloc_mutex);
    NoallocDevice &d = noalloc_dev[dev];
    if (!d.ready) {
        void *ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, noalloc_scratch);
        if (e == cudaSuccess && (ptr == nullptr || ((uintptr_t)ptr & 255u))) e = cudaErrorInvalidSymbol;
        if (e != cudaSuccess) return e;
        int L = 512;
        for (int i = 0; i < 5 && e == cudaSuccess; ++i, L *= 2) { FDAS_DISPATCH_L(L, (e = noalloc_prepare<LL>(dev, &d.grid_max[i]))); }
        if (e != cudaSuccess) return e;
        d.base = (unsigned char *)ptr;
        d.ready = true;
    }
    *out = &d;
    return cudaSuccess;
}

} // namespace

extern "C" fdas_status fdas_convolve_noalloc(int64_t n_f, int n_batch, int z_max, int z_step, int template_width, int segment_len,
                                             const float *d_templates, const void *d_spectrum, float *d_power, void *cuda_stream)
{
    // the argument rules of fdas_plan_create / fdas_plan_set_batch / fdas_convolve
    if (n_f < 1 || n_batch < 1 || z_max < 0 || z_step < 1 || (z_max % z_step) != 0) return FDAS_ERR_INVALID_ARG;
    if (template_width < 2 || (template_width & 1)) return FDAS_ERR_INVALID_ARG;
    if (segment_len < 2 || (segment_len & (segment_len - 1))) return FDAS_ERR_INVALID_ARG;
    if (!supported_L(segment_len)) return FDAS_ERR_UNSUPPORTED;
    if (template_width > segment_len / 2) return FDAS_ERR_INVALID_ARG;
    if (!d_templates || !d_spectrum || !d_power) return FDAS_ERR_INVALID_ARG;
    if (((uintptr_t)d_templates & 7u) || ((uintptr_t)d_spectrum & 7u) || ((uintptr_t)d_power & 3u)) return FDAS_ERR_INVALID_ARG;
    const int L = segment_len, m = template_width;
    const int64_t n_z = 2 * (int64_t)(z_max / z_step) + 1;
    // the one limit of this entry point: the transformed bank has to fit its part of the static array
    if (n_z * (int64_t)L > (int64_t)FDAS_NOALLOC_MAX_BANK) return FDAS_ERR_TOO_LARGE;

    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return FDAS_ERR_CUDA; }
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return FDAS_ERR_UNSUPPORTED;
    const NoallocDevice *d = nullptr;
    e = noalloc_device(dev, &d);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return FDAS_ERR_CUDA; }

    unsigned int *work = (unsigned int *)(d->base + NOALLOC_WORK_OFF);
    float2 *tw = (float2 *)(d->base + NOALLOC_TW_OFF);
    float4 *bank = (float4 *)(d->base + NOALLOC_BANK_OFF);
    cudaStream_t st = (cudaStream_t)cuda_stream;

    // (1) twiddle table of this L, counters to zero
    fdas_noalloc_init_kernel<<<(L + 255) / 256, 256, 0, st>>>(tw, L, work);
    e = cudaGetLastError();
    // (2) the bank: conj, pad, 1/L, forward transform, register order (fdas_set_templates' kernel, on the caller's stream)
    if (e == cudaSuccess) {
        e = cudaErrorInvalidValue;
        FDAS_DISPATCH_L(L, (e = noalloc_bank<LL>((const float2 *)d_templates, m, (int)n_z, tw, bank, st)));
    }
    // (3) the hot kernel, as fdas_convolve launches it
    if (e == cudaSuccess) {
        ConvParams cp;
        cp.spectrum = (const float2 *)d_spectrum;
        cp.power = d_power;
        cp.amp = nullptr;
        cp.bmax = nullptr;
        cp.barg = nullptr;
        cp.gperm = bank;
        cp.tw = tw;
        cp.work = work;
        cp.n_f = n_f;
        cp.S = L - m;
        cp.n_seg = (n_f + cp.S - 1) / cp.S;
        cp.n_work = cp.n_seg * (int64_t)n_batch;
        cp.w_begin = 0;
        cp.n_z = (int)n_z;
        cp.m = m;
        cp.bulk_ok = ((uintptr_t)d_spectrum & 15u) == 0;
        const int gmax = d->grid_max[noalloc_L_index(L)];
        e = cudaErrorInvalidValue;
        FDAS_DISPATCH_L(L, (e = launch_convolve<LL, OUT_POWER>(cp, gmax, st)));
    }
    if (e != cudaSuccess) { (void)cudaGetLastError(); return FDAS_ERR_CUDA; }
    return FDAS_OK;
}

extern "C" {

// The kernel generation is what profiles/traffic.json is keyed by: bump it with every change to the hot kernel.
const char *fdas_version(void) { return "libfdas sm_100a k8"; }

} // extern "C"

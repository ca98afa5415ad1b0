/*
 * fdas.h -- C ABI of libfdas.so: the FDAS matched-filter hot path on one B200 (sm_100a).
 *
 * What the library computes (arXiv:1711.10855; P:NN = line NN of the paper text, PAPER.md):
 *
 *   eq.(2), P:21-23   A'_{r0} = sum_k A_k conj(H_{r0-k})   "correlating the m bins around bin r0 with
 *                     the predicted, normalized, Fourier response H", for every acceleration trial z,
 *   P:31 (section 2)  evaluated by overlap-and-save: the spectrum is cut into segments of length L,
 *                     each is Fourier transformed on chip (eq.(3)), multiplied by the
 *                     transformed template of every z, inverse transformed, trimmed of its aliased
 *                     part and merged "in such a way as to produce the linear convolution",
 *   BASELINE.json     and written as the float32 power plane P[z][r0] = |A'_{r0}|^2.
 *
 * With the template of trial z given as m taps h_z[j], tap j <-> offset d = j - m/2 (DESIGN.md,
 * readings 1, 6, 7):
 *
 *   P[b][i][r0] = | sum_{j=0}^{m-1} A[b][r0 + m/2 - j] * conj(h_i[j]) |^2 ,   A[b][k] := 0 for k outside [0, n_f)
 *
 * for batch item b < n_batch, template row i < n_z (row i <-> z = -z_max + i*z_step), column r0 < n_f.
 * All arithmetic is IEEE float32 (FMA contraction allowed); the result equals the definition up to
 * rounding.  There is no CPU fallback: every entry point that needs the GPU fails with FDAS_ERR_CUDA
 * if none is usable.
 *
 * Conventions: "HOST" / "DEVICE" say where a pointer must live.  Complex data are interleaved
 * (re, im) float32 pairs.  No exception crosses this boundary; no global state (one exception: the static device
 * scratch of fdas_convolve_noalloc, described there); a plan may be used from several host threads as long as
 * calls on the same plan are not concurrent (the asynchronous launches fdas_convolve, fdas_convolve_complex and
 * fdas_detect_blockmax are the exception: see fdas_convolve).
 */
#ifndef FDAS_H
#define FDAS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fdas_plan fdas_plan; /* opaque; owned by the library between create and destroy */

typedef enum {
    FDAS_OK = 0,
    FDAS_ERR_INVALID_ARG = 1,  /* NULL pointer, bad size, misaligned buffer */
    FDAS_ERR_UNSUPPORTED = 2,  /* segment_len not in {512, 1024, 2048, 4096, 8192} */
    FDAS_ERR_ALLOC = 3,        /* host or device allocation failed */
    FDAS_ERR_NO_TEMPLATES = 4, /* fdas_convolve before fdas_set_templates */
    FDAS_ERR_CUDA = 5,         /* a CUDA runtime call failed; see fdas_plan_last_cuda_error */
    FDAS_ERR_TOO_LARGE = 6     /* fdas_convolve_noalloc: n_z * segment_len exceeds FDAS_NOALLOC_MAX_BANK */
} fdas_status;

/*
 * Create a plan for spectra of n_f bins, trials z = -z_max, -z_max+z_step, ..., +z_max
 * (n_z = 2*z_max/z_step + 1), templates of template_width = m taps and overlap-and-save segments of
 * segment_len = L points (argument list from BASELINE.json north_star).  The plan keeps
 * S = L - m outputs per segment (any step <= L-m+1 gives the same linear convolution, P:31;
 * DESIGN.md reading 8) and n_seg = ceil(n_f / S) segments per spectrum.  Batch count starts at 1.
 *
 *   out            HOST, receives the plan; untouched on error
 *   n_f            >= 1
 *   z_max, z_step  z_max >= 0, z_step >= 1, z_max % z_step == 0
 *   template_width even, >= 2, <= segment_len / 2
 *   segment_len    512, 1024, 2048, 4096 or 8192 (else FDAS_ERR_UNSUPPORTED)
 *
 * Allocates plan-owned device memory on the current CUDA device: the transformed template bank
 * (n_z * L complex64) and a twiddle table (L complex64, eq.(3)).
 */
fdas_status fdas_plan_create(fdas_plan **out, int64_t n_f, int z_max, int z_step,
                             int template_width, int segment_len);

/* Number of independent spectra one fdas_convolve call processes (BASELINE.json config 5:
 * "64 independent spectra ... computed in one fdas_convolve call").  n_batch >= 1.  Templates are
 * shared by all batch items.  Cheap; may be called between convolves. */
fdas_status fdas_plan_set_batch(fdas_plan *plan, int n_batch);

/*
 * Give the plan its template bank ("predicted, normalized, Fourier response H").
 *   h_templates   HOST, float32 [n_z][m][2] (re, im); row i <-> z = -z_max + i*z_step; tap j <-> offset
 *                 j - m/2.  Copied during the call; the caller may free it afterwards.
 * The library conjugates the taps (eq.(2): conj(H)), zero-pads to L, scales by 1/L (the inverse
 * transform's factor, reading 9), transforms them with its own FFT kernel and stores the
 * spectra in the register order the convolution kernel reads.  Synchronous: returns after the
 * device work has finished.  May be called again to replace the bank: the call first waits for
 * the whole device (cudaDeviceSynchronize), so work still reading the old bank finishes first.
 */
fdas_status fdas_set_templates(fdas_plan *plan, const float *h_templates);

/*
 * The FDAS-specific optimisation the paper mentions ("exploit symmetries in FDAS algorithm"): the
 * response of trial -z is the complex conjugate of the response of +z, so P[-z](A) = P[+z](conj A) and one
 * template fetch can serve two rows (SURVEY.md 8(c) note S).  enable != 0 asks
 * fdas_convolve to use that form WHEN it is exact: fdas_set_templates checks that row n_z-1-i of the bank is the
 * element-wise conjugate of row i bit for bit (n_z odd); any other bank, and segment lengths other than 2048 and
 * 4096, silently take the general path.  Off by default: measured slower than the general path on
 * BASELINE.json config 3 (profiles/r2_symmetry.md).  fdas_plan_symmetry_active tells which path the next
 * fdas_convolve takes.  The result is the same to rounding (tests/test_gpu_symmetry.py).
 */
fdas_status fdas_plan_set_symmetry(fdas_plan *plan, int enable);
int fdas_plan_symmetry_active(const fdas_plan *plan);

/*
 * Enqueue the hot path on cuda_stream: for every batch item, segment and trial z -- segment load,
 * forward FFT (once per segment), pointwise multiply, inverse FFT, trim, |.|^2, power-plane write.
 *   d_spectrum    DEVICE, complex64 [n_batch][n_f], read only, 8-byte aligned (16-byte alignment lets interior
 *                 segments be staged by the bulk-copy engine; otherwise they are loaded with plain loads)
 *   d_power       DEVICE, float32 [n_batch][n_z][n_f], written completely, 4-byte aligned (128-byte
 *                 alignment and n_f % 32 == 0 give fully coalesced line writes; rows 32 bytes off the line
 *                 grid cost 0.5 %, rows 4 bytes off 3.3 % on config 3: profiles/r2_c3_k7.md)
 *   cuda_stream   a cudaStream_t passed as void* (NULL = the legacy default stream)
 * Asynchronous: only launches; never synchronises, allocates or copies.  The buffers must stay
 * valid until the stream has run the work.  Output is bitwise reproducible (the kernel hands out
 * segments through an atomic counter, but which CTA computes a segment does not change its result).
 * The plan may be used from several streams at once, also from several host threads (one stream each; the
 * counter hand-out is atomic); at most 1024 launches of one plan may be in flight (enqueued and not finished)
 * at any time: they take the plan's work counters round robin.  fdas_plan_last_launch_count then reports on
 * whichever call wrote last.
 * Must be called with the plan's device current (the one current at fdas_plan_create).
 * Errors: INVALID_ARG (NULL / misaligned pointers), NO_TEMPLATES, CUDA (launch failure).
 */
fdas_status fdas_convolve(fdas_plan *plan, const void *d_spectrum, float *d_power, void *cuda_stream);

/*
 * fdas_convolve for callers that must not allocate device memory: the whole of fdas_plan_create +
 * fdas_set_templates + fdas_convolve in one call that never calls cudaMalloc, cudaFree or any routine that does.
 *
 * Who needs it.  Every other way into this library goes through a plan, and a plan is built from cudaMalloc calls
 * (the transformed bank, the twiddle table, the work counters; fdas_set_templates adds a temporary).  Some hosts
 * cannot afford that: a telescope back end that carved up the whole card when it started and keeps searching for
 * days, where a cudaMalloc in the middle of the run stalls every stream of the device while the driver maps memory
 * and can fail outright because nothing is left; a process in which a framework's pool allocator already holds
 * the free memory, so the driver has none to give although the pool has plenty; code that is handed its buffers
 * and is forbidden by its own rules to take more (fixed memory budgets, certification, a callback that runs while
 * other work is in flight).  Such a caller passes its inputs and its output as usual, and the memory the kernels
 * need besides them comes out of the library image instead.
 *
 * Where the scratch lives.  libfdas.so carries one file-scope __device__ array of FDAS_NOALLOC_SCRATCH_BYTES
 * (8 MiB + 64 KiB + 256 B).  The CUDA runtime gives every GPU that loads the library its own copy when the
 * library's device code is loaded there and keeps it until the process exits, whether this entry point is ever
 * called or not.  It holds, in this order, the two work counters of the persistent kernel, the twiddle table
 * w_L^j (eq.(3); 8192 entries at most) and the transformed template bank (n_z * L complex64).  The bank is
 * what sets THE LIMIT: n_z * segment_len <= FDAS_NOALLOC_MAX_BANK = 2^20 elements, enough for every
 * BASELINE.json configuration (config 3: 201 * 4096 = 823 296).  A larger request is refused with
 * FDAS_ERR_TOO_LARGE before anything is launched; use a plan for those.
 *
 * What a call does, all on cuda_stream and in this order: (1) one small kernel writes the twiddle table for this
 * segment_len and sets the work counters to zero; (2) the template kernel of fdas_set_templates conjugates, pads,
 * scales and transforms the taps into the scratch bank; (3) the hot kernel of fdas_convolve runs exactly as it does
 * for a plan.  Nothing is kept between calls on purpose: the array still holds whatever the previous call left
 * (another bank, the table of another segment length, counters of a launch that was aborted), so every call
 * rewrites all of what it reads and clears the counters itself.  The price is the template transform on every
 * call, n_z of the (1 + n_z) * n_seg transforms -- 0.1 % on config 3.
 *
 *   n_f, z_max, z_step, template_width, segment_len   as fdas_plan_create (same checks, same errors)
 *   n_batch       >= 1, as fdas_plan_set_batch
 *   d_templates   DEVICE, float32 [n_z][m][2] as in fdas_set_templates but already on the GPU, 8-byte aligned,
 *                 read only (the caller owns it; a host pointer here faults inside the kernel)
 *   d_spectrum, d_power, cuda_stream   as fdas_convolve
 * Asynchronous.  The result equals fdas_convolve's to rounding (the twiddle table is evaluated on the GPU here and
 * on the host there; the two could differ in the last bit of an entry -- on the shapes of
 * tests/test_zz_no_alloc.py they do not, and the planes agree bit for bit).
 *
 * All calls on one GPU share the one array.  Two calls whose GPU work overlaps -- different streams, or different
 * host threads -- overwrite each other's bank and counters and both results are garbage without any error being
 * reported: put them on one stream or order them with events.  Calls on different GPUs are independent.
 *
 * First call on each GPU: besides the above it looks up the device address of the array (cudaGetSymbolAddress,
 * with that GPU current) and raises the kernels' shared-memory limits (cudaFuncSetAttribute).  These are host-side
 * set-up calls, not stream work.  Make this first call before you begin any stream capture on that GPU.
 * Thread safe with respect to that set-up; at most 64 GPUs per process (more: FDAS_ERR_UNSUPPORTED).
 * Errors: INVALID_ARG, UNSUPPORTED, TOO_LARGE as described (all three are decided before the first CUDA call);
 * CUDA if the set-up or a launch fails (the runtime's error state has been cleared by then; there is no plan to
 * ask for the code).
 */
#define FDAS_NOALLOC_MAX_BANK (1 << 20)                                   /* complex64 elements: n_z * segment_len */
#define FDAS_NOALLOC_SCRATCH_BYTES (256 + 8 * 8192 + 8 * FDAS_NOALLOC_MAX_BANK)
fdas_status fdas_convolve_noalloc(int64_t n_f, int n_batch, int z_max, int z_step, int template_width, int segment_len,
                                  const float *d_templates, const void *d_spectrum, float *d_power, void *cuda_stream);

/*
 * Convenience for callers whose data live in HOST memory (bench.py's "e2e" leg): copies
 * h_spectrum to a plan-owned device buffer, runs fdas_convolve, copies the power plane back to
 * h_power, and synchronises the stream.  On an error return, too, nothing is left in flight that touches
 * h_spectrum or h_power (the call waits for what it had enqueued): the caller may free them at once.  Buffers are allocated on first use and kept by the plan:
 * two *_host calls on one plan must not overlap (not from two host threads, not on two streams).
 *   h_spectrum    HOST (pinned memory gives asynchronous copies), complex64 [n_batch][n_f]
 *   h_power       HOST, float32 [n_batch][n_z][n_f]
 */
fdas_status fdas_convolve_host(fdas_plan *plan, const void *h_spectrum, float *h_power, void *cuda_stream);

/*
 * The paper's general convolution ("produce the linear convolution", Table 2): the same path,
 * but the filtered spectrum A' of eq.(2) itself is stored instead of its power.
 *   d_amp         DEVICE, complex64 [n_batch][n_z][n_f], written completely, 8-byte aligned
 * Otherwise as fdas_convolve (asynchronous, same errors).
 */
fdas_status fdas_convolve_complex(fdas_plan *plan, const void *d_spectrum, void *d_amp, void *cuda_stream);

/*
 * The hot path fused with the first step of detection ("detect"; "FDAS code"; the paper leaves the
 * detection stage to Dimoudi et al. 2017, so this one is defined here, reading 17): the power plane is
 * never written.  The columns are cut into n_blk = fdas_plan_nseg(plan) blocks of blk = fdas_plan_step(plan)
 * columns, block s = [s*blk, min((s+1)*blk, n_f)), and for every batch item b, template row i and block s
 *   d_max[b][i][s] = max over the block of P[b][i][r0]                  (float32, the value the plane would hold)
 *   d_arg[b][i][s] = the smallest r0 - s*blk that attains it             (int32, 0 <= . < blk)
 *   d_max, d_arg  DEVICE, [n_batch][n_z][n_blk], 4-byte aligned, written completely
 * Comparisons are made on the float32 powers; equal powers resolve to the lowest column.  Deterministic.
 * Otherwise as fdas_convolve (asynchronous, same errors).  fdas_detect_blockmax_host is the HOST-pointer
 * convenience (spectrum in, the two small arrays out; synchronises the stream), like fdas_convolve_host; when the
 * call is several waves of work it uploads the spectrum in up to 8 pieces on a plan-owned copy stream and launches
 * each piece's segments as it arrives, so that most of the host-to-device copy hides behind the kernel.
 */
fdas_status fdas_detect_blockmax(fdas_plan *plan, const void *d_spectrum, float *d_max, int32_t *d_arg, void *cuda_stream);
fdas_status fdas_detect_blockmax_host(fdas_plan *plan, const void *h_spectrum, float *h_max, int32_t *h_arg, void *cuda_stream);

/*
 * Detection down to a candidate list ("detect", "FDAS code"; reading 20): fdas_detect_blockmax
 * followed by a threshold on the block maxima.  A block maximum is a candidate iff its float32 power is >= threshold
 * (inclusive); the list is ordered by (item, row, column), which makes it unique, and holds at most `capacity` entries:
 *   d_cand        DEVICE, fdas_candidate [capacity], 4-byte aligned; entries [0, d_count[1]) are written, the rest is
 *                 left untouched
 *   d_count       DEVICE, int32 [2]: d_count[0] = number of candidates found (all of them, may exceed capacity: then
 *                 the list holds the first `capacity` in order and d_count[0] - d_count[1] were dropped);
 *                 d_count[1] = number written = min(found, capacity)
 *   threshold     float32 power (templates of unit norm on whitened noise give a mean power of 2)
 *   capacity      >= 0; n_batch * n_z * n_blk must be < 2^31
 * The block maxima go to a plan-owned scratch buffer (8 bytes per (item, row, block) + 4 per row), allocated by the
 * first call on the plan and when n_batch has grown since: that call allocates, later ones only launch (the hot kernel
 * and three small ones).  Deterministic, no atomics.  One such call per plan at a time (they share the scratch).
 * Otherwise as fdas_convolve (asynchronous, same errors, plus FDAS_ERR_ALLOC).  fdas_detect_candidates_host takes the
 * spectrum from HOST memory and returns both results to HOST memory (h_cand [capacity], h_count [2]; 16 * capacity + 8
 * bytes come back whatever the count, so entries of h_cand at and beyond h_count[1] are unspecified), uploads like fdas_detect_blockmax_host, and synchronises the stream.
 */
typedef struct {
    int32_t item;    /* batch item */
    int32_t row;     /* template row i <-> z = -z_max + i * z_step */
    int32_t column;  /* r0 of the block maximum */
    float power;     /* the float32 value the power plane would hold there */
} fdas_candidate;
fdas_status fdas_detect_candidates(fdas_plan *plan, const void *d_spectrum, float threshold, int capacity,
                                   fdas_candidate *d_cand, int32_t *d_count, void *cuda_stream);
fdas_status fdas_detect_candidates_host(fdas_plan *plan, const void *h_spectrum, float threshold, int capacity,
                                        fdas_candidate *h_cand, int32_t *h_count, void *cuda_stream);

/*
 * The segment FFT as a stand-alone batched transform (eq.(3); the stand-alone comparison of P:46 and
 * Table 1: "100 FFTs per kernel launch, while launching 1000 of these kernels", N = 1024, with the
 * number of elements per thread as the design axis).  Same device code as the convolution kernel's forward
 * transform; natural order in and out.
 *   n                 512, 1024, 2048, 4096 or 8192 (else FDAS_ERR_UNSUPPORTED)
 *   elems_per_thread  0 = the convolution kernel's choice; 8 (n = 512, 1024) or 16 (n >= 1024); other
 *                     combinations are FDAS_ERR_UNSUPPORTED
 * fdas_fft_exec enqueues one launch that transforms n_fft contiguous sequences:
 *   d_in, d_out       DEVICE, complex64 [n_fft][n], 8-byte aligned, must not overlap
 *   inverse           0: eq.(3);  1: the unnormalised inverse (conjugate twiddles)
 * Asynchronous; never allocates or synchronises.  Errors as fdas_convolve.
 */
typedef struct fdas_fft_plan fdas_fft_plan;
fdas_status fdas_fft_plan_create(fdas_fft_plan **out, int n, int elems_per_thread);
fdas_status fdas_fft_exec(fdas_fft_plan *plan, int64_t n_fft, const void *d_in, void *d_out, int inverse, void *cuda_stream);
/* The repetition scheme of P:46: n_launches launches of n_fft transforms each, enqueued back to back.  Launch i
 * transforms sequences [i*n_fft, (i+1)*n_fft), so d_in and d_out are DEVICE complex64 [n_launches * n_fft][n] and the
 * 1000 x 100 protocol reads and writes 100 000 distinct sequences (from and to HBM), the same data as one launch of
 * 100 000.  From 8 launches on, the launches are recorded once as a CUDA graph (the same kernels; as they touch
 * disjoint sequences the graph orders launch i only after launch i-4, four chains that may overlap on the GPU) and
 * the graph is launched on cuda_stream, in order with the stream's other work: the first call with a given argument set
 * does that host-side work (milliseconds) and allocates the graph; calls repeating the last argument set only launch it.
 * One call per plan at a time. */
fdas_status fdas_fft_exec_many(fdas_fft_plan *plan, int n_launches, int64_t n_fft, const void *d_in, void *d_out,
                               int inverse, void *cuda_stream);
fdas_status fdas_fft_plan_destroy(fdas_fft_plan *plan);
int fdas_fft_plan_elems_per_thread(const fdas_fft_plan *plan);
int fdas_fft_plan_grid(const fdas_fft_plan *plan);   /* CTAs of one launch at most (grid-stride over the batch) */

/*
 * The step before the correlation ("the FFT output of the observation"; reading 18): the real
 * time series of n_samples float32 samples -> its n_samples/2 lowest Fourier bins (eq.(3)), whitened.
 *   n_samples     a power of two, 2^19 .. 2^27 (else FDAS_ERR_UNSUPPORTED); BASELINE.json config 3: 2^23
 *   whiten_block  > 0: bins are cut into blocks of that many bins, block b = [b*blk, min((b+1)*blk, n/2)), and every
 *                 block is scaled by sqrt(2 / mean |X_k|^2) (bin 0 counted as 0 and set to 0) so that re and im
 *                 have unit variance where the block is noise; a block of zeros stays zero.  <= 0: not whitened.
 *   d_series      DEVICE, float32 [n_samples], 8-byte aligned, read only
 *   d_spectrum    DEVICE, complex64 [n_samples/2] -- what fdas_convolve takes as d_spectrum
 * fdas_spectrum_exec enqueues six launches on the stream (three transposes, two batched segment FFTs, one
 * separate-and-whiten pass) using two plan-owned scratch buffers of n_samples/2 complex64: one exec of a plan at a
 * time.  Asynchronous; deterministic.
 */
typedef struct fdas_spectrum_plan fdas_spectrum_plan;
fdas_status fdas_spectrum_plan_create(fdas_spectrum_plan **out, int64_t n_samples, int64_t whiten_block);
fdas_status fdas_spectrum_exec(fdas_spectrum_plan *plan, const float *d_series, void *d_spectrum, void *cuda_stream);
fdas_status fdas_spectrum_plan_destroy(fdas_spectrum_plan *plan);
int64_t fdas_spectrum_plan_bins(const fdas_spectrum_plan *plan);  /* n_samples / 2 */

/* Free the plan and everything it owns.  NULL is accepted. */
fdas_status fdas_plan_destroy(fdas_plan *plan);

/* Plan geometry (0 / -1 on NULL). */
int fdas_plan_nz(const fdas_plan *plan);            /* n_z */
int fdas_plan_step(const fdas_plan *plan);          /* S = outputs kept per segment */
int64_t fdas_plan_nseg(const fdas_plan *plan);      /* segments per spectrum */
int fdas_plan_batch(const fdas_plan *plan);         /* n_batch */
int fdas_plan_grid(const fdas_plan *plan);          /* CTAs of the persistent hot kernel: resident CTAs per SM x SMs */

/* Number of kernel launches the last fdas_convolve on this plan made (bench.py "gpu_launches"). */
int fdas_plan_last_launch_count(const fdas_plan *plan);

/* cudaError_t of the last failing CUDA call on this plan (0 if none), and its text. */
int fdas_plan_last_cuda_error(const fdas_plan *plan);
const char *fdas_status_string(fdas_status s);

/*
 * Debug / test entry: forward FFT (eq.(3)) of n_seg contiguous length-L segments with the
 * same device code the hot path uses, returned in NATURAL frequency order.
 *   d_in, d_out   DEVICE, complex64 [n_seg][L]; must not overlap
 *   inverse       0: eq.(3);  1: the unnormalised inverse (conjugate twiddles)
 * Synchronous.  Used by tests/ to check the segment FFT against the oracle's brute-force DFT.
 */
fdas_status fdas_debug_fft(int segment_len, int64_t n_seg, const void *d_in, void *d_out, int inverse);

/*
 * Debug / test entry (HOST only, no GPU needed): evaluates the index maps of the inverse transform
 * of the hot loop exactly as the kernels do (same functions, compiled for the host), so that the
 * layout logic -- which element a thread register holds, the shuffle register permutation, the
 * shared-memory addresses of the exchanges and the twiddle-table indices -- can be checked on a CPU.
 *   what = FDAS_LAYOUT_GEOMETRY  a selects: 0 P (passes), 1 E (elements/thread), 2 NT (threads),
 *          3 Ra, 4 Rb (radices of the first two inverse passes), 5 Gs (shuffle group), 6 NA, 7 NB,
 *          8 elements of one exchange buffer, 9 R0, 10 R1
 *   FDAS_LAYOUT_FREQ      natural frequency index held by register a*Ra + b of thread t at loop entry
 *   FDAS_LAYOUT_GMOD      index j: the template spectrum element of register (., a) is stored times conj(w_L^j)
 *   FDAS_LAYOUT_TWA       index j: register a*Rb + b is multiplied by conj(w_L^j) before the second pass
 *   FDAS_LAYOUT_FIX       index j: thread t's outputs equal the exact inverse DFT times conj(w_L^j)
 *   FDAS_LAYOUT_SHFL_SRC / _DST  register sent / written in shuffle round a for the pair b = i*NA + j
 *   FDAS_LAYOUT_WRITE_A   shared-memory element written from register a*Rb + b (first exchange)
 *   FDAS_LAYOUT_READ_A    shared-memory element read into register a*R + b   (R = R0 if P == 3, else R1)
 *   FDAS_LAYOUT_WRITE_B / _READ_B  second exchange (P == 4 only): register a*R1 + b / register a
 *   FDAS_LAYOUT_TW_MID    (P == 4) index j: register (., a) of the third pass is multiplied by conj(w_L^j)
 * w_L = exp(-2 pi i / L).  Returns -1 for arguments out of range or an unsupported segment_len.
 */
enum {
    FDAS_LAYOUT_GEOMETRY = 0, FDAS_LAYOUT_FREQ = 1, FDAS_LAYOUT_GMOD = 2, FDAS_LAYOUT_TWA = 3, FDAS_LAYOUT_FIX = 4,
    FDAS_LAYOUT_SHFL_SRC = 5, FDAS_LAYOUT_SHFL_DST = 6, FDAS_LAYOUT_WRITE_A = 7, FDAS_LAYOUT_READ_A = 8,
    FDAS_LAYOUT_WRITE_B = 9, FDAS_LAYOUT_READ_B = 10, FDAS_LAYOUT_TW_MID = 11
};
int64_t fdas_debug_layout(int segment_len, int what, int t, int a, int b);

/*
 * Measurement support (bench.py --mode peak): the FP32 FMA rate this GPU reaches on register-only chains of
 * dependent FMAs, scalar (packed = 0) or packed FFMA2 (packed = 1), in TFLOP/s by CUDA events.  It is what the
 * nominal "alu" peak of the roofline (SMs x 128 lanes x 2 x max clock) is checked against.  Synchronous.
 */
fdas_status fdas_debug_alu_peak(int packed, double *tflops_out, double *ms_out);

/* Library build info: e.g. "libfdas sm_100a <date>".  Never NULL. */
const char *fdas_version(void);

#ifdef __cplusplus
}
#endif
#endif /* FDAS_H */

/*
 * plspec.h -- C ABI of the B200-native plasma-line spectral integrator.
 *
 * One operation (arXiv 2311.18737, "GPGPU Acceleration of Incoherent Scatter Radar Plasma
 * Line Analysis"; citations are PAPER.md line numbers + section):
 *
 *   for every inter-pulse period (IPP) p and range gate r
 *       d[t]    = V[p][r0 + r*stride + t] * conj(C[p][t])   t <  code_len   (sec. 3.2.1)
 *               = 0                                          code_len <= t < N
 *       X[f]    = sum_{t<N} d[t] * exp(-2*pi*i*f*t/N)                         (sec. 3.2.2)
 *       S[r][f] += |X[f]|^2 = Re^2 + Im^2                                     (Eq. 8, 113-115 sec. 3.2.3)
 *   summed over every IPP given since create / the last finalize             (sec. 3.2.4)
 *
 * Un-normalised forward FFT, plain sum over IPPs (no 1/N, no 1/P), natural bin order with
 * DC at f = 0.  All arithmetic runs in fp32 CUDA kernels (sm_100a); there is no CPU path.
 *
 * Conventions
 *   - Every function returns an int status: PLSPEC_OK (0) or a negative PLSPEC_ERR_*.
 *     Nothing is printed, thrown or aborted across this boundary.
 *   - Pointers marked [host] are host pointers; [device] are CUDA device pointers on the
 *     device that was current at plspec_create; [host|device] may be either (detected with
 *     cudaPointerGetAttributes).
 *   - The caller owns every buffer it passes.  The library owns the handle and everything
 *     behind it (accumulators, tables, staging buffers, streams) until plspec_destroy.
 *   - A handle is not thread-safe; distinct handles are independent.
 */
#ifndef PLSPEC_H
#define PLSPEC_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct plspec_ctx *plspec_handle;   /* opaque, library-owned */

/* dtype of `voltages` (codes are always interleaved float32 re,im). */
enum { PLSPEC_CF32 = 0,    /* interleaved float32 (re, im), 8 bytes / sample                    */
       PLSPEC_SC16 = 1 };  /* interleaved little-endian int16 (I, Q), 4 bytes / sample, converted
                              exactly on the device, NO 1/32768 scaling (S is in counts^2)      */

enum { PLSPEC_OK = 0,
       PLSPEC_ERR_INVALID_ARG = -1,  /* bad argument; no state changed                          */
       PLSPEC_ERR_ALLOC       = -2,  /* host or device allocation failed                        */
       PLSPEC_ERR_CUDA        = -3,  /* a CUDA call failed; see plspec_last_cuda_error          */
       PLSPEC_ERR_UNSUPPORTED = -4 };/* valid request this build cannot serve (e.g. not sm_100) */

/* plspec_configure options (EXTENSION; defaults in brackets). */
enum { PLSPEC_OPT_KERNEL     = 1,   /* [0] 0 = auto, 1 = generic radix-2 kernel, 2 = fused kernel   */
       PLSPEC_OPT_IPP_CHUNKS = 2,   /* [0] fused kernel: 0 = one CTA per SM, each an equal contiguous run of the
                                       launch's (gate group, IPP) work items; else each gate group's IPPs are split
                                       into this many equal runs, one CTA each.  Partial sums of a gate meet in S
                                       through fp32 atomic adds either way.                               */
       PLSPEC_OPT_H2D_BATCH  = 3,   /* [0] 0 = auto; IPPs per host->device staging batch            */
       PLSPEC_OPT_BPSK_PACK  = 4,   /* [1] 1 = a pre-pass kernel bit-packs the codes of each accumulate when every
                                       sample is exactly +-1+0j (binary phase codes) and the fused kernel decodes
                                       by sign flip; any other code takes the general complex decode.
                                       0 = always decode generally.  Results are identical either way.   */
       PLSPEC_OPT_STAGE      = 5, /* [1] 1 = the fused kernel prefetches each IPP's samples into shared memory
                                       with bulk asynchronous copies whenever the run of samples one CTA needs
                                       fits (N <= 16384 and, for complex64 input, N <= 8192); 0 = it always
                                       loads voltages straight from global memory.  Results are identical.  */
       PLSPEC_OPT_SPLIT      = 6,   /* [1] N > 16384 only: how the N/16384 residues of a window (each its own
                                       length-16384 transform, held by its own CTA) get the decoded samples.
                                       1 = scratch: a pre-pass kernel writes every decoded window (with the outer
                                       radix-N/16384 butterfly) to a device buffer (<= 4 GiB, IPPs batched to fit),
                                       the fused kernel reads it back.  2 = ring: one cooperative launch; every CTA
                                       decodes a slice of all windows of the current step into a ring of
                                       PLSPEC_OPT_RING_DEPTH steps that stays in L2, and transforms its residue
                                       from there (no DRAM traffic for the decoded windows; measured slower than 1
                                       on B200).  0 = each (gate, residue) CTA decodes the whole
                                       window itself (no scratch, N/16384 times the loads).  Results agree to
                                       rounding.                                                                 */
       PLSPEC_OPT_SHARED_CODE = 7,  /* [0] 1 = `codes` of plspec_accumulate holds ONE code of code_len samples that
                                       decodes every IPP of the call (a transmitter that repeats its waveform, e.g.
                                       the chirp of BASELINE config 4); 0 = codes[n_ipp][code_len], one per IPP.
                                                                                            */
       PLSPEC_OPT_DEFER      = 8,   /* [1] host-buffer calls only.  1 = the second half of each call's IPPs is copied
                                       to the device at once but transformed later: by plspec_finalize, one gate
                                       range after the other, so that each range's spectra are written out (device
                                       -> host) while the next range is still being transformed; or, if another
                                       plspec_accumulate comes first, by that call.  0 = every IPP is transformed
                                       by the call that brought it.  Results are identical.                       */
       PLSPEC_OPT_RING_DEPTH = 9,   /* [3] 2..16: steps the ring of PLSPEC_OPT_SPLIT = 2 holds (148 x 128 KB each)     */
       PLSPEC_OPT_RING_AHEAD = 10   /* [2] 1..depth-1: steps a slice is decoded ahead of its use                       */
     };

/* Counters since create (EXTENSION; used by bench.py for gpu_launches / h2d bytes). */
typedef struct {
    long long kernel_launches;   /* kernels of this library launched                       */
    long long h2d_bytes;         /* bytes copied host->device by plspec_accumulate          */
    long long d2h_bytes;         /* bytes copied device->host by plspec_finalize            */
    long long ipps_accumulated;  /* IPPs accumulated since create                           */
    int       kernel_kind;       /* 1 = generic, 2 = fused (what `auto` resolved to)        */
    int       ipp_chunks_last;   /* IPP chunks per gate used by the last accumulate (0 = balanced runs) */
} plspec_stats_t;

/*
 * Create an integrator.  ("iterating through the number of range gates we desire
 * and the amount to step each of them"; "4096 range gates with a step size of 25,
 * starting at the first element"; PAPER.md:111 power-of-two row length.)
 *   N         FFT length, a power of two in [16, 65536]
 *   code_len  samples per transmit code, 1 <= code_len <= N (shorter codes are zero-padded to N)
 *   n_ranges  number of range gates R >= 1
 *   r0        first sample of gate 0 within an IPP, >= 0
 *   stride    samples between successive gates, >= 1
 *   ipp_len   EXTENSION: samples per IPP row of `voltages` (the pitch); 0 means the tightly
 *             packed span r0 + (R-1)*stride + code_len.  The span must fit in ipp_len.
 *   dtype     PLSPEC_CF32 or PLSPEC_SC16
 *   out       [host] receives the handle; NULL on any error
 * Allocates S_dev[R][N] fp32 on the current device (zeroed) and the twiddle tables.
 */
int plspec_create(int N, int code_len, int n_ranges, int r0, int stride, int ipp_len,
                  int dtype, plspec_handle *out);

/*
 * Accumulate n_ipp pulses: S[r][f] += |FFT_N(decode(p, r))[f]|^2 for every gate r.
 *   voltages  [host|device] voltages[n_ipp][ipp_len], element per dtype, C-contiguous
 *   codes     [host|device] codes[n_ipp][code_len], interleaved float32 (re, im); one code per
 *             IPP ("a single full TX and echo" per pulse)
 *   n_ipp     >= 0; 0 is a successful no-op
 *   stream    cudaStream_t to order the work on (NULL = the legacy default stream)
 * Device pointers: the fused kernel is enqueued on `stream` and the call returns without
 * synchronising; the buffers must stay valid until that stream work completes.
 * Host pointers: the needed span of each IPP (not the whole row: PAPER.md:149 item 3) and its
 * code are copied in batches on an internal copy stream, overlapped with compute on `stream`
 * (PAPER.md:149 item 2).  Pinned buffers make the copies asynchronous; they must stay valid
 * until plspec_finalize (or a synchronisation of `stream`).  Pageable buffers work but the
 * copies are staged synchronously by the driver.  Both pointers must be of the same kind.
 */
int plspec_accumulate(plspec_handle h, const void *voltages, const void *codes,
                      int n_ipp, void *stream);

/*
 * Finish an integration: wait for all accumulate work, write S_out[n_ranges][N] (fp32,
 * row-major, natural FFT bin order, un-normalised sum) and zero the accumulators so the next
 * integration starts clean ("Upon completion, we transfer the spectrum result
 * back").  S_out is [host|device]; the call blocks until S_out is complete.  The work is enqueued on the stream of the
 * latest plspec_accumulate (plspec_reset and plspec_finalize_products likewise): that stream must still exist.
 * Host S_out: the deferred pulses of a host-buffer call (PLSPEC_OPT_DEFER) are transformed here, one gate range after
 * the other, and each finished range is copied out while the next one computes; pinned memory makes those copies
 * asynchronous.
 */
int plspec_finalize(plspec_handle h, float *S_out);

/*
 * EXTENSION (the step after the hot path): per range gate of a finished spectrum,
 * where the plasma lines are.  PAPER.md:40-45 (Eq. 1): the plasma line lies at +-f_r from the ion line, and
 * f_r follows the electron density with range; PAPER.md:79 (Eq. 8): the estimate is the AVERAGE power.
 *   S         [device] S[n_ranges][N] as written by plspec_finalize (sum over n_ipp pulses, natural bin order),
 *             16-byte aligned
 *   n_ipp     pulses summed in S (>= 1): reported powers are S / n_ipp
 *   k_min     1 <= k_min < N/2: bins |f| < k_min (DC and the ion line) are left out
 *   guard     >= 0: bins within `guard` of either line are left out of the noise floor
 *   k_up      [device] int[n_ranges]: arg max of S over k_min <= f < N/2 (up-shifted line, +f_r)
 *   k_dn      [device] int[n_ranges]: arg max over N/2 < f <= N - k_min (down-shifted line, bin N - f_r);
 *             the lowest bin wins a tie in both
 *   p_up,p_dn [device] float[n_ranges]: S / n_ipp at those bins
 *   noise     [device] float[n_ranges]: mean of S / n_ipp over the other bins of [k_min, N - k_min] \ {N/2}
 *   stream    cudaStream_t; one kernel is enqueued and the call returns without synchronising
 * Caller owns every buffer.  Errors: PLSPEC_ERR_INVALID_ARG (null or host pointer, S misaligned, N not a power of two
 * in [16, 65536], range errors), PLSPEC_ERR_CUDA.  Needs no handle.
 */
int plspec_profile(const float *S, int n_ranges, int N, int n_ipp, int k_min, int guard,
                   int *k_up, float *p_up, int *k_dn, float *p_dn, float *noise, void *stream);

/*
 * EXTENSION: plspec_profile for callers that cannot allocate device memory (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc).  Same arguments, same five outputs (k_up, p_up, k_dn, p_dn equal
 * plspec_profile's bit for bit; noise to float64 summation order, ~1e-7 relative), computed by a (gate, column tile)
 * grid whose CTAs meet in a 32-byte workspace per gate.  That workspace is a file-scope array in device memory
 * (csrc/plspec_static.cu) of PLSPEC_STATIC_MAX_GATES entries: 256 KiB that every GPU which loads the library holds
 * until the process exits.  The call makes no cudaMalloc / cudaFree and calls no allocating library routine; it
 * enqueues one memset (clearing the entries it uses) and one kernel on `stream` and returns without synchronising.
 *   n_ranges  1 ... PLSPEC_STATIC_MAX_GATES; more is PLSPEC_ERR_INVALID_ARG (use plspec_profile)
 * All calls, on every stream and from every thread, SHARE the one workspace of the device: two calls that overlap
 * on the GPU race on it and their outputs are undefined.  Calls on one stream, or ordered by events, are safe.
 * Errors: as plspec_profile, plus PLSPEC_ERR_UNSUPPORTED (device is not sm_100).  Needs no handle.
 */
#define PLSPEC_STATIC_MAX_GATES 8192
int plspec_profile_static(const float *S, int n_ranges, int N, int n_ipp, int k_min, int guard,
                          int *k_up, float *p_up, int *k_dn, float *p_dn, float *noise, void *stream);

/*
 * EXTENSION ("mean P = S/P (Eq. 8), optional fftshift"): the mean power spectrum of a
 * finished integration, PAPER.md:79 (Eq. 8: the estimate is the AVERAGE <|x|^2>; the hot path keeps the plain
 * sum, reading A2), optionally with zero frequency moved to the middle of every row.
 *   S         [device] S[n_ranges][N] as written by plspec_finalize, 16-byte aligned
 *   P_out     [device] float[n_ranges][N], 16-byte aligned, must not alias S:
 *             P_out[r][g] = S[r][f] / n_ipp (one IEEE float32 division), with g = f when centred = 0 and
 *             g = (f + N/2) mod N when centred = 1 (DC at column N/2, negative frequencies to its left)
 *   n_ipp     pulses summed in S (>= 1); 1 gives the plain (shifted) copy
 *   stream    cudaStream_t; one kernel is enqueued and the call returns without synchronising
 * Caller owns both buffers.  Errors: PLSPEC_ERR_INVALID_ARG (null, host, misaligned or aliased pointer, N not a
 * power of two in [16, 65536], n_ranges < 1, n_ipp < 1, centred not 0/1), PLSPEC_ERR_CUDA.  Needs no handle.
 */
int plspec_mean_spectrum(const float *S, float *P_out, int n_ranges, int N, int n_ipp, int centred, void *stream);

/*
 * EXTENSION (the row-wise products "fuse into finalize"): plspec_finalize to DEVICE memory
 * with the products of plspec_mean_spectrum and / or plspec_profile computed in the same pass over the accumulators,
 * while each gate's bins are being put into natural order -- S is read once; S_out and P_out are written once.
 * Same definitions and the same results as the two stand-alone calls applied to S_out (line bins, powers and mean
 * spectrum bit for bit; the noise floor to float64 summation order).
 */
typedef struct {
    int    n_ipp;     /* pulses summed since the last finalize (>= 1): the divisor of Eq. 8's average  */
    int    centred;   /* P_out: 0 = natural bin order, 1 = zero frequency at column N/2                             */
    float *P_out;     /* [device] float[n_ranges][N], 16-byte aligned, or NULL: no mean spectrum                   */
    int    k_min;     /* line search: 1 <= k_min < N/2 (see plspec_profile)                                         */
    int    guard;     /* line search: >= 0                                                                          */
    int   *k_up;      /* [device] int[n_ranges]   \                                                                 */
    float *p_up;      /* [device] float[n_ranges]  |  all five, or all NULL: no line search                         */
    int   *k_dn;      /* [device] int[n_ranges]    |                                                                */
    float *p_dn;      /* [device] float[n_ranges]  |                                                                */
    float *noise;     /* [device] float[n_ranges] /                                                                 */
} plspec_products_t;
/*
 *   S_out  [device] float[n_ranges][N], 16-byte aligned: the un-normalised sum, as plspec_finalize writes it
 *   prod   [host]   what else to compute; the struct is read during the call only
 * Blocks until everything is written; zeroes the accumulators.  Errors: PLSPEC_ERR_INVALID_ARG (null handle / S_out /
 * prod, host or misaligned pointers, P_out == S_out, some but not all line-search outputs, range errors),
 * PLSPEC_ERR_CUDA.
 */
int plspec_finalize_products(plspec_handle h, float *S_out, const plspec_products_t *prod);

/*
 * DIAGNOSTIC ("measured FMA peak to be reported beside" the derived one): the
 * FP32 multiply-add issue rate of the current device, the measured denominator of the path's ALU roofline
 * (5 N log2 N flop per decoded window).  Launches reps + 1 kernels of 4 x 512 threads per SM, each
 * thread running 32 independent multiply-add chains for `iters` iterations (64 flop per thread and iteration; no
 * memory traffic), times each with CUDA events on `stream` and blocks until done.
 *   packed       0 = scalar FFMA, 1 = packed FFMA2 (two lanes per instruction: the form the fused kernel issues)
 *   iters        >= 1 loop iterations per thread (1 << 16 gives launches of a few milliseconds)
 *   reps         1 ... 100000 timed launches after one warm-up launch
 *   tflops_best  [host] fastest launch, in TFLOP/s (2 flop per multiply-add)
 *   tflops_mean  [host] mean over the `reps` launches (sustained rate when reps spans seconds)
 * Errors: PLSPEC_ERR_INVALID_ARG, PLSPEC_ERR_ALLOC, PLSPEC_ERR_CUDA.  Needs no handle; touches no integrator state.
 */
int plspec_diag_fp32_peak(int packed, int iters, int reps, double *tflops_best, double *tflops_mean, void *stream);

/*
 * DIAGNOSTIC (the N > 16384 paths): streaming bandwidth of the current device with 128-bit
 * accesses, the figures behind the scratch-versus-ring argument.  `n_ctas` CTAs of 512 threads each walk a buffer of
 * `bytes` bytes (allocated and freed by the call, rounded down to whole MiB) `passes` times; one warm-up launch, then
 * the fastest of three launches, timed with CUDA events on `stream`; the call blocks.  A buffer well below the L2 size
 * (126 MB on B200) measures the SM <-> L2 paths, a buffer of gigabytes DRAM.
 *   kind   0 = read (ld.global.cg), 1 = write (st.global), 2 = copy first half -> second half (bytes read + written
 *          are counted), 3 = write by the TMA engine (cp.async.bulk stores of 16 KB from shared memory, 4 in flight)
 *   bytes  1 MiB ... 8 GiB;  n_ctas 1 ... 65535 (148 = one per SM);  passes >= 1
 *   gbs    [host] bandwidth in GB/s
 * Errors: PLSPEC_ERR_INVALID_ARG, PLSPEC_ERR_ALLOC, PLSPEC_ERR_CUDA.  Needs no handle.
 */
int plspec_diag_mem_bandwidth(int kind, long long bytes, int n_ctas, int passes, double *gbs, void *stream);

/* EXTENSIONS ------------------------------------------------------------------------------- */
int plspec_reset(plspec_handle h);                        /* zero the accumulators, no output */
int plspec_destroy(plspec_handle h);                      /* free everything; NULL is OK       */
int plspec_configure(plspec_handle h, int option, int value);
int plspec_get_stats(plspec_handle h, plspec_stats_t *out /* [host] */);
int plspec_last_cuda_error(plspec_handle h);              /* cudaError_t of the last failure   */
const char *plspec_strerror(int status);                  /* static string, never NULL         */
const char *plspec_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PLSPEC_H */

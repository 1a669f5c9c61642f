/* spiir.h -- C ABI of the B200-native SPIIR template-bank filter.
 *
 * Operation (BASELINE.json:north_star; section 3.1 "a parallel bank of single pole IIR
 * filters", section 3.3 "parameter array and the detection data within given time window
 * ... output data of each filter which is the input data in the next iteration", L329/L339 "The SNR of
 * one template needs the outputs of all its filters ... sum all the output"):
 *
 *     y_{t,k}[n] = a1_{t,k} * y_{t,k}[n-1] + b0_{t,k} * x[n - d_{t,k}]
 *     SNR_t[n]   = sum_k y_{t,k}[n]
 *
 * a1, b0 complex, d integer >= 0, x real (whitened strain).  All arithmetic is FP32 on the GPU.
 * Semantics fixed at this boundary: zero initial state y[-1] = 0; zero
 * pre-history x[m<0] = 0; d = 0 is the current sample; the sample index is global across calls; the
 * output is the plain sum (no normalisation); the order of a template's filters does not matter
 * (up to rounding).  The summation order is fixed by the bank layout, so results are bitwise
 * reproducible from run to run and independent of a template's position in the bank.
 *
 * Every step of the path runs in the library's own CUDA kernels (sm_100a).  There is no CPU fallback:
 * without a CUDA device every call that needs one fails with SPIIR_ECUDA.
 *
 * Threading and streams: a handle is not thread-safe; distinct handles are.  Work is enqueued on the caller's
 * stream and is ordered with respect to it.  The calls that touch a bank's state (spiir_filter, spiir_filter_peaks,
 * spiir_filter_host[_async], spiir_bank_reset, spiir_bank_get_state, spiir_bank_set_state) are also ordered among
 * themselves in the order they are issued, whatever streams they name: a call that arrives on another stream than
 * its predecessor makes its stream wait for an event recorded behind the predecessor's work (so alternating streams is
 * safe, and costs one event per switch; calls that stay on one stream put nothing between their kernels).  The
 * caller's own buffers (x_dev, snr_dev, ...) are ordered only by the stream they are used on.
 * Host synchronisation and allocation: calls return without synchronising the host, except
 *   - spiir_bank_create / spiir_bank_destroy (synchronise the device),
 *   - spiir_filter_host and spiir_bank_host_sync (by contract),
 *   - spiir_filter / spiir_filter_peaks when n exceeds every earlier call AND the 65 536 samples the input tape is
 *     created for: the tape is then reallocated (cudaMalloc + one stream synchronisation),
 *   - the first streaming-path call (one cudaMalloc of the per-tile scratch) and the first spiir_filter_peaks (one
 *     cudaMalloc of [T] keys),
 *   - spiir_filter_peaks with snr_dev == NULL on a bank with templates of more than 8 warp tiles, whenever n exceeds
 *     every earlier such call (private SNR rows are reallocated: cudaMalloc + one stream synchronisation),
 *   - spiir_filter_host_async when n exceeds every earlier call (staging buffers are reallocated).
 * Every call makes the bank's device current for its duration and restores the caller's current device on return.
 */
#ifndef SPIIR_H
#define SPIIR_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct spiir_bank spiir_bank; /* opaque; owns device coefficients, filter state, input history */

enum {
    SPIIR_OK = 0,
    SPIIR_EINVAL = -1, /* bad argument (null, negative, inconsistent sizes, non-finite, |a1| >= 1) */
    SPIIR_ENOMEM = -2, /* host or device allocation failed */
    SPIIR_ECUDA = -3,  /* CUDA runtime / launch error, or no usable device */
    SPIIR_ESTATE = -4  /* handle unusable (a previous call failed part-way) */
};

/* Kernel path used by spiir_filter (north_star subsystems (3) and (4)). */
enum {
    SPIIR_PATH_AUTO = 0,       /* choose per call from bank size and chunk length */
    SPIIR_PATH_THROUGHPUT = 1, /* filters across lanes, sequential in time, smem-staged window */
    SPIIR_PATH_SCAN = 2,       /* time-parallel: segments per filter + linear-recurrence carry scan */
    SPIIR_PATH_STREAM = 3      /* tiny chunks, many filters (set at create): calls of <= 64 samples run as independent
                                  warps + an ordered combine pass, one sweep over coefficients and state per call;
                                  longer calls on the same bank use the blocked kernel */
};

typedef struct spiir_options {
    int32_t struct_size;        /* = sizeof(spiir_options); lets the struct grow compatibly */
    int32_t path;               /* SPIIR_PATH_*; default AUTO */
    int32_t filters_per_thread; /* 0 = choose; else 1, 2, 4, 8 or 16 (register blocking of the throughput kernel) */
    int32_t scan_segments;      /* 0 = choose; else time segments per call for SPIIR_PATH_SCAN */
    int32_t warps_per_cta;      /* 0 = choose; else 8, 16 or 32; valid (filters_per_thread, warps_per_cta) pairs:
                                   (16,8) (8,8) (8,16) (4,8) (4,16) (4,32) (2,32) (1,32).  spiir_bank_create returns
                                   SPIIR_EINVAL for any other pair; when only one of the two is given the other follows
                                   it.  SPIIR_PATH_STREAM banks use 8 warps unless told otherwise, hence
                                   filters_per_thread 4, 8 or 16 there */
    int32_t window_copies;      /* 0 = choose; else 1, 2 or 4 shifted copies of the input window in shared memory
                                   (= floats per shared-memory load); falls back if they do not fit */
    int32_t small_templates;    /* templates of <= 16 x filters_per_thread filters sharing warp tiles (sub-warp segments of 4,
                                   8 or 16 lanes): 0 = choose, 1 = on, 2 = off.  Shared tiles exist
                                   for the blockings (8,16), (4,16) and (2,32); the cheapest for the bank is taken unless
                                   filters_per_thread / warps_per_cta name one.  Not used with SPIIR_PATH_STREAM. */
    int32_t scan_launches;      /* kernel launches per call of the two low-latency paths.  0 = choose: SPIIR_PATH_SCAN takes
                                   one cooperative launch when every CTA of the items x segments grid is resident (else
                                   three), SPIIR_PATH_STREAM a tile kernel + a combine kernel chained by programmatic
                                   dependent launch (measured faster than one launch).  1 = one launch wherever the
                                   grid can meet at a barrier (both paths; the streaming kernel is then a plain launch of
                                   at most SMs x occupancy CTAs that spin at a grid-wide barrier: do not run it beside
                                   other kernels that keep SMs occupied indefinitely).  3 = always separate kernels (scan: carry
                                   pass, carry scan, output pass).  All forms of a path give the same bits.  Any other
                                   value is SPIIR_EINVAL */
} spiir_options;

/* Build a bank.  All pointers are HOST pointers; the arrays are copied, the caller keeps ownership.
 *   n_templates      T >= 1
 *   filter_offsets   [T+1] CSR offsets into the filter arrays, offsets[0] = 0, strictly increasing
 *                    (every template has >= 1 filter); K = offsets[T]
 *   a1, b0           [2K] float32, (re, im) interleaved = complex64; |a1| < 1 and everything finite
 *   delays           [K] int32, d >= 0
 *   device           CUDA device ordinal
 *   opt              nullable (defaults)
 * The bank lays the filters out on the device in structure-of-arrays form, each template's filters
 * sorted by delay, dealt to lanes so that a warp's shared-memory reads of x[n-d] avoid bank
 * conflicts, and padded with null filters (a1 = b0 = 0) to the kernel's tile size (north_star
 * subsystem (1); "aligned and continuous").  State and history start at zero.
 * Synchronises the host with the device.  On error *out is NULL. */
int spiir_bank_create(spiir_bank **out, int32_t n_templates, const int64_t *filter_offsets,
                      const float *a1, const float *b0, const int32_t *delays, int32_t device,
                      const spiir_options *opt);

/* Filter the next n samples of strain.
 *   x_dev     DEVICE pointer, [n] float32, caller-owned
 *   snr_dev   DEVICE pointer, complex64 as (re, im) float32 pairs; row t starts at snr_dev + 2*t*ld;
 *             exactly SNR[t][0..n) is written for every template t, nothing else is touched
 *   ld        row stride in complex elements, ld >= n (lets chunked calls fill columns of one [T][N] buffer)
 *   stream    cudaStream_t (NULL = legacy default stream)
 * n = 0 is a no-op.  Any n >= 1 and any sequence of chunk sizes is valid, including n smaller than the
 * largest delay.  Carries filter state y and the last max_delay input samples to the next call.
 * Enqueues on the stream and returns; x_dev and snr_dev must stay valid until the stream reaches
 * that point.  SPIIR_EINVAL on null pointers, n < 0 or ld < n; SPIIR_ECUDA on launch failure. */
int spiir_filter(spiir_bank *bank, const float *x_dev, int64_t n, float *snr_dev, int64_t ld,
                 void *stream);

/* Filter the next n samples like spiir_filter and reduce them to one trigger candidate per template (SURVEY.md
 * NEXT N4; "rapidly detect ... signals" -- the paper defines no trigger, reading Q16):
 *   power_dev[t] = max over the n samples of this call of |SNR_t[j]|^2   (float32, computed from the FP32 SNR)
 *   index_dev[t] = the first j in 0..n-1 that attains it
 * Both DEVICE [T]; either may be NULL.  snr_dev may be NULL: then the series itself is not written (the only
 * per-sample HBM traffic of the path disappears).  n >= 1.  The maximum is merged with integer atomic max
 * over (power bits, index), so the result does not depend on the order of execution. */
int spiir_filter_peaks(spiir_bank *bank, const float *x_dev, int64_t n, float *snr_dev, int64_t ld,
                       float *power_dev, int32_t *index_dev, void *stream);

/* spiir_filter for callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): one tiny-chunk call of a bank created with SPIIR_PATH_STREAM, same arguments, same results (the same two
 * kernels; bitwise equal to spiir_filter), but the per-tile partial sums go to a file-scope device array of the library
 * instead of a buffer from cudaMalloc.  The call reaches no cudaMalloc, cudaFree or allocating library routine.
 *   limits   n <= 64 samples; the bank has at most 8192 warp tiles (32 x filters_per_thread filter slots each: 1 048 576
 *            slots at the streaming default of 4 filters per thread); the array is 4 MiB and every GPU that loads the
 *            library holds it until exit.  Anything beyond returns SPIIR_EINVAL with a message saying which limit;
 *            so does a call that would have to create an event (a bank moved to another stream for the first time).
 *   set-up   the first call on a device looks the array's address up (cudaGetSymbolAddress) and sets the kernel's
 *            attributes: make it before a graph capture starts.
 *   sharing  all banks and calls on a device share the array, which keeps the last call's contents.  Nothing has to start
 *            at zero (every row the combine pass reads is written by the tile pass of the same call), but calls that
 *            overlap on the GPU -- two banks on different streams -- race on it: serialise them.
 * May be mixed with spiir_filter on the same bank (state and history carry over either way). */
int spiir_filter_static(spiir_bank *bank, const float *x_dev, int64_t n, float *snr_dev, int64_t ld,
                        void *stream);

/* Same operation with HOST buffers (the end-to-end entry): copies x to the device, filters, copies
 * SNR[t][0..n) back into snr_host (row stride ld), overlapping copies and kernels internally.
 * Buffers may be pageable or pinned.  Returns after the results are in snr_host. */
int spiir_filter_host(spiir_bank *bank, const float *x_host, int64_t n, float *snr_host, int64_t ld);

/* The same, but returns as soon as the work is enqueued on the bank's own streams: the copies of this chunk's
 * results overlap the kernels of the next chunk ("overlapping technology").  x_host and snr_host
 * must be PINNED host memory and stay untouched until spiir_bank_host_sync returns; calls may be issued back to
 * back (they are ordered).  spiir_bank_host_sync blocks until every enqueued chunk's results are in host memory. */
int spiir_filter_host_async(spiir_bank *bank, const float *x_host, int64_t n, float *snr_host, int64_t ld);
int spiir_bank_host_sync(spiir_bank *bank);

/* Zero the filter state and the input history (a cold bank again); enqueued on the stream.  Waits first for chunks
 * of spiir_filter_host_async that are still in flight. */
int spiir_bank_reset(spiir_bank *bank, void *stream);

/* Sizes.  Return -1 for a null handle. */
int64_t spiir_bank_num_templates(const spiir_bank *bank);
int64_t spiir_bank_num_filters(const spiir_bank *bank); /* real filters K, padding excluded */
int64_t spiir_bank_max_delay(const spiir_bank *bank);   /* D = max_k d_k = length of the carried history */

/* Checkpoint / resume.  y_dev: DEVICE [2K] float32 (re, im) in the CALLER's filter order;
 * hist_dev: DEVICE [D] float32, hist[j] = x[n_done - D + j] (oldest first).  Either may be NULL to skip it. */
int spiir_bank_get_state(spiir_bank *bank, float *y_dev, float *hist_dev, void *stream);
int spiir_bank_set_state(spiir_bank *bank, const float *y_dev, const float *hist_dev, void *stream);

/* Free everything the bank owns (synchronises the device).  NULL is a no-op. */
int spiir_bank_destroy(spiir_bank *bank);

/* Host-only diagnostic (no CUDA call): lay the bank out exactly as spiir_bank_create would for the given
 * register blocking (filters_per_thread F in {1,2,4,8,16}, warps_per_cta W: a valid pair, see spiir_options;
 * window_copies NC in {1,2,4}) and
 * report it.  slot_of_filter (nullable, [K] int64, HOST) receives the device slot of every caller filter;
 * stats (nullable, [8] double, HOST) receives {n_slots, n_warp_tiles, n_cta_items, n_rounds,
 * avg_conflict_degree (mean over load phases of the largest number of lanes on one bank group; 1 = conflict
 * free), padding_fraction = 1 - K/n_slots, uniform_groups (1 if every warp position always belongs to the
 * same template shape, which enables per-template barriers), segmented (1 if small templates share tiles)}.
 * pack_small != 0 lays templates of <= 16 * filters_per_thread filters out in shared tiles as spiir_bank_create does
 * with small_templates = 1.  Same argument checks as spiir_bank_create. */
int spiir_layout_probe(int32_t n_templates, const int64_t *filter_offsets, const int32_t *delays,
                       int32_t filters_per_thread, int32_t warps_per_cta, int32_t window_copies,
                       int64_t *slot_of_filter, double *stats, int32_t pack_small);

/* Introspection. */
const char *spiir_last_error(void);      /* thread-local message of the last failing call */
int64_t spiir_kernel_launches(void);     /* kernels this library has launched in this process */
int32_t spiir_bank_last_path(const spiir_bank *bank); /* SPIIR_PATH_* used by the last spiir_filter */
int32_t spiir_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SPIIR_H */

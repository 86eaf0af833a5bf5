/*
 * fengine.h -- C ABI of the B200-native F-engine (channelizer) data path.
 *
 * The path is the one stated in arxiv 2303.09886 Sec. 2.1:
 *   1. unpack 10-bit signed samples
 *   2. integer coarse delay as an index offset
 *   3. T-tap polyphase FIR, Eq. (1)
 *        g[t] = sum_{j<T} s[N*m - c + t + N*j] * w[t][j],  N = 2n
 *   4. N-point real-to-complex FFT, keep the n non-negative channels, drop Nyquist
 *   5. fine delay: X[k] * exp(i(-2 pi d k / N + phi))
 *   6. complex per-channel gain
 *   7. quantise to 8-bit signed Gaussian integers, both polarisations interleaved
 *      (PAPER.md:43, :45, :161): round-half-even, clamp to [-127, 127].
 * Call names and argument lists follow BASELINE.json:north_star; everything else is this build's
 * choice (DESIGN.md section 2 lists the readings R1..R18).
 *
 * Conventions
 *   - plain C, no torch types; "host" / "device" is stated for every pointer.
 *   - every function returning int returns a FENGINE_* status; nothing is thrown across the ABI.
 *   - a handle is not thread-safe and is driven from ONE CUDA stream at a time (its scratch and tables are
 *     shared by all calls): order calls on different streams yourself (events) or use one handle per stream.
 *     Independent handles are independent.  A handle belongs to the device that was current at create; calls
 *     made with another current device fail with FENGINE_ERR_STATE.
 *   - setters copy their host arrays before returning (caller keeps ownership) and take effect
 *     for later fengine_process calls.  They rebuild the derived tables and synchronise the device before
 *     AND after (off the hot path), so a later call on any stream, blocking or not, sees the new values;
 *     fengine_process itself never launches a table kernel.
 *   - there is no CPU fallback: without a CUDA device every call fails with FENGINE_ERR_CUDA.
 */
#ifndef FENGINE_H
#define FENGINE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fengine fengine_t;   /* opaque; one per engine (group of antennas sharing weights) */

enum {
    FENGINE_OK = 0,
    FENGINE_ERR_INVALID_ARG = 1,    /* bad size / null pointer / non-finite parameter */
    FENGINE_ERR_ALLOC = 2,          /* host or device allocation failed */
    FENGINE_ERR_CUDA = 3,           /* a CUDA call failed (see fengine_last_error) */
    FENGINE_ERR_STATE = 4           /* tables too short for the requested n_spectra */
};

/*
 * fengine_create -- one antenna (an F-engine is the pipeline for the two
 * polarisations of one antenna).  Same as fengine_create_batched(1, ...).
 *
 * n_channels  n, a power of two, 8 <= n <= 32768 (1024, 4096, 8192, 32768).
 * taps        T, 1 <= T <= 32 (PAPER.md:39: up to 16; :245 measures 32).  T = 2, 4, 8, 16 run the tiled kernels for
 *             n >= 1024; T = 32 runs them on the pol-packed path (n_pols = 2, n <= 8192, equal coarse delays in
 *             both pols); every other shape runs the generic one-thread-per-output kernels (slow, for tests).
 * n_pols      1 or 2.
 * weights     HOST, N*T floats, N = 2n, flat time order weights[t + N*j] = w[t][j] of Eq. (1)
 *             (BASELINE.json configs[0]).  Must be finite.  Copied.
 * Returns NULL on failure (invalid argument, no device, allocation failure).
 * Defaults after create: coarse delay 0, fine delay 0, phase 0, gain 1.
 */
fengine_t *fengine_create(int n_channels, int taps, int n_pols, const float *weights);

/* n_antennas >= 1 antennas sharing the weights; antenna is the outermost index of in / out. */
fengine_t *fengine_create_batched(int n_antennas, int n_channels, int taps, int n_pols,
                                  const float *weights);

void fengine_destroy(fengine_t *fe);

/*
 * Coarse delays (Eq. (1) index t0 + t - c + 2nj): c in samples, may be negative
 * or larger than N.  Positive c reads earlier samples.
 * c             HOST int32 [A][P][n_per_stream].
 * n_per_stream  1 = one value per stream for the whole call; otherwise entry m applies to spectrum
 *               m of a fengine_process call and n_per_stream must be >= that call's n_spectra.
 * Samples whose index falls outside [0, L) read as 0 (R3).
 */
int fengine_set_coarse_delays(fengine_t *fe, const int32_t *c, int64_t n_per_stream);

/*
 * Fine delays: channel k is multiplied by exp(i(-2 pi delay k / N + phase)),
 * delay in samples, phase in radians (BASELINE.json configs[0]).
 * delay, phase  HOST float [A][P][n_per_stream], same n_per_stream rule as above.  Must be finite.
 */
int fengine_set_fine_delays(fengine_t *fe, const float *delay, const float *phase,
                            int64_t n_per_stream);

/*
 * Bandpass gains.
 * gains_re_im   HOST float [A][P][n][2] (re, im).  Must be finite.
 */
int fengine_set_gains(fengine_t *fe, const float *gains_re_im);

/*
 * fengine_process -- the hot path, steps 1-7 for n_spectra spectra of every stream.
 *
 * in         DEVICE, 16-byte aligned, [A][P][L*5/4] bytes, L = N*(n_spectra + T - 1) samples per
 *            stream: 10-bit two's complement, big-endian bit stream (sample u in bits
 *            [10u, 10u+10), MSB first, BASELINE.json configs[0]).
 * out        DEVICE, 16-byte aligned, [A][n_spectra][n][P][2] int8 (re, im).
 * n_spectra  S >= 0 (0 is a no-op).
 * stream     a cudaStream_t (NULL = default stream).
 * Enqueues kernels on `stream` and returns without synchronising; never touches host memory and
 * never allocates (scratch is sized at create / first call with a larger S -- see DESIGN.md).
 * Spectrum m of stream (a, p) starts at sample N*m - c[a][p][m] (R2).
 */
int fengine_process(fengine_t *fe, const void *in, void *out, int64_t n_spectra, void *stream);

/*
 * fengine_reserve -- size every buffer fengine_process needs for calls of up to max_spectra spectra (SURVEY.md 8(b):
 * "the library never allocates in this call").  Without a reserve the first fengine_process call, and any call larger
 * than all before it, allocates (and synchronises the device once); after a successful reserve fengine_process never
 * allocates, never synchronises, and can be captured in a CUDA graph: a call that would need more returns
 * FENGINE_ERR_STATE.  The reserve is made for the kernels the handle would run now (options, equal or unequal
 * coarse delays of the two pols); call it again after changing those.  Off the hot path: synchronises the device.
 */
int fengine_reserve(fengine_t *fe, int64_t max_spectra);

/*
 * fengine_process_host -- the same path for HOST buffers (the paper's regime: input chunks arrive
 * in pinned host memory and results go back to the host).
 * in_host / out_host  HOST pointers (pinned or pageable), same layouts as fengine_process.
 * Copies the input to device staging owned by the handle (grown on first use), runs the path on an
 * internal stream, copies the result back and synchronises before returning.  On the tiled two-kernel path the
 * call is cut into "host_chunks" pieces of spectra (option, default 8) and the upload of the rows a piece needs,
 * its kernels and the download of its output records run on three streams, so that PCIe is busy in both
 * directions under the kernels (the paper's chunked pipeline); pinned host buffers are needed
 * for the copies to overlap.  The result is identical to fengine_process on the same data.
 */
int fengine_process_host(fengine_t *fe, const void *in_host, void *out_host, int64_t n_spectra);

/*
 * fengine_process_heaps -- the same path with the output in the channel-major heaps the X-engines consume
 * ("each heap contains data for 256 spectra ... a c x 256 x 2 array of Gaussian integers";
 * the post-processing transposes from time-major to channel-major within each heap).
 * in         DEVICE, as fengine_process.
 * heaps_out  DEVICE, 16-byte aligned, [A][ceil(S / 256)][n][256][P][2] int8: heap h of antenna a holds spectra
 *            256 h .. 256 h + 255, channel-major; spectra past S in the last heap are written as zero.
 * The time-major records are produced by the kernels of fengine_process into a buffer owned by the handle (sized
 * at the first call) and transposed through shared memory by one more kernel; n >= 32.
 */
int fengine_process_heaps(fengine_t *fe, const void *in, void *heaps_out, int64_t n_spectra, void *stream);

/*
 * Streaming (the input is processed in chunks and the samples a chunk's last spectra still need
 * are carried over to the next chunk; coarse delays reach outside the chunk).  Between
 * fengine_stream_begin and fengine_stream_end consecutive fengine_stream_push calls continue ONE sample stream per
 * (antenna, pol): every call supplies the next n_new rows of N samples and returns n_new spectra; the handle keeps
 * the rows that later windows still need in a device window buffer (two buffers, tail copied device to device).
 *
 * fengine_stream_begin   sizes the history from the coarse delays set so far: D = T - 1 + ceil(max(-c, 0) / N) rows of
 *                        latency (written to *delay_out if non-null) and ceil(max(c, 0) / N) + 1 further rows of
 *                        history; max_new_spectra bounds n_new of every push.  Samples before the first push are 0.
 * fengine_stream_push    in_new: DEVICE, 16-byte aligned, [A][P][n_new * N * bits / 8] bytes (the new rows only);
 *                        out: DEVICE [A][n_new][n][P][2] int8.  Output j of the push is spectrum G + j - D of the
 *                        stream, G = rows pushed before this call: the concatenated outputs of all pushes equal
 *                        fengine_process on [D zero rows, then the whole stream] (same coarse delays), which is what
 *                        the tests check.  Delay tables with n_per_stream > 1 are indexed by j.  Coarse delays set
 *                        during a stream must not need more history than begin kept (FENGINE_ERR_STATE).
 * fengine_stream_end     closes the stream; fengine_process is refused while one is open.
 */
int fengine_stream_begin(fengine_t *fe, int64_t max_new_spectra, int64_t *delay_out);
int fengine_stream_push(fengine_t *fe, const void *in_new, void *out, int64_t n_new, void *stream);
int fengine_stream_end(fengine_t *fe);

/*
 * fengine_process_noalloc -- steps 1-7 in one call that allocates nothing, for callers that cannot
 * call cudaMalloc: programs that gave the whole GPU to their own memory pool at start-up, real-time receive loops
 * that cannot take the device-wide stall of an allocation, hosts that forbid allocation after
 * initialisation.  There is no handle (creating one allocates): every table is a DEVICE pointer the caller owns, and
 * the FIR -> transform intermediate lives in a fixed array built into the library (FENGINE_NOALLOC_MAX_FLOATS floats =
 * 4 MiB of device memory, held by every GPU that loads the library until the process exits).
 *
 * in             DEVICE [A][P][L*5/4] bytes, 10-bit samples as fengine_process, L = N*(n_spectra + taps - 1), N = 2n.
 * out            DEVICE [A][n_spectra][n][P][2] int8, as fengine_process.
 * weights        DEVICE float [N*taps], weights[t + N*j] = w[t][j] of Eq. (1).
 * coarse_delays  DEVICE int32 [A][P], one value per stream for the whole call.
 * fine_delays, phases  DEVICE float [A][P].
 * gains_re_im    DEVICE float [A][P][n][2], 8-byte aligned.
 * n_channels     n, a power of two in [8, 32768]; taps 1..32; n_pols 1 or 2; n_antennas >= 1; n_spectra >= 0.
 * stream         a cudaStream_t (NULL = default stream); kernels are enqueued, the call does not synchronise.
 * err, err_len   HOST buffer for a message when the return value is not FENGINE_OK (may be NULL / 0).
 *
 * Limit: A * P * n_spectra * N <= FENGINE_NOALLOC_MAX_FLOATS (e.g. 128 spectra of one dual-pol antenna at n = 2048);
 * a larger call is refused with FENGINE_ERR_INVALID_ARG and a message that states the limit -- split the batch.
 * The caller's tables are read as they are at kernel run time and are not validated (non-finite values propagate).
 * Runs the simple one-thread-per-output kernels (the "force_generic" path of fengine_process), so the result is that
 * path's; it is not the fast path.
 * First call on a device: looks up the device address of the built-in array (once per device; no allocation).  Make
 * that first call with the device current and before any stream capture begins.
 * All calls on a device share the array, which keeps the previous call's contents (every word that is read is written
 * first by the same call, so nothing needs clearing).  Calls whose kernels may overlap on the GPU -- two streams with no
 * event between them, two host threads -- race on it: serialise them.
 */
#define FENGINE_NOALLOC_MAX_FLOATS (1 << 20)
int fengine_process_noalloc(const void *in, void *out, const float *weights, const int32_t *coarse_delays,
                            const float *fine_delays, const float *phases, const float *gains_re_im,
                            int n_antennas, int n_channels, int taps, int n_pols, int64_t n_spectra,
                            void *stream, char *err, int64_t err_len);

/* Human-readable description of the last error on this handle ("" if none). */
const char *fengine_last_error(const fengine_t *fe);

/* ---- test hooks: same kernels, intermediate results exposed (tolerances are stated on them) ---- */

/* Pre-quantisation spectra Y (after rotation and gain): DEVICE float [A][n_spectra][n][P][2]. */
int fengine_process_f32(fengine_t *fe, const void *in, float *spectra_out, int64_t n_spectra,
                        void *stream);

/* Unpacked, coarse-delayed window samples: DEVICE int16 [A][P][n_spectra][N*T] (small cases only):
 * element i of spectrum m is s[N*m - c + i] (0 outside the batch).  Bit-exact check of steps 1-2.
 * This hook runs a one-thread-per-sample SIDE kernel that no timed configuration launches; the unpackers of the
 * kernels fengine_process runs are checked bit-exactly through fengine_debug_fir with one-hot weights (fir_kernel,
 * fir2_kernel, fir3_kernel) and, where the rows never leave the chip as integers (split producer, pipelined kernel),
 * through fengine_process_f32 with one-hot weights (tests/test_gpu_parity.py). */
int fengine_debug_unpack(fengine_t *fe, const void *in, int16_t *samples_out, int64_t n_spectra,
                         void *stream);

/* FIR output g of Eq. (1) in natural column order: DEVICE float [A][P][n_spectra][N].  Runs the FIR kernel of the path
 * fengine_debug_path reports for pol_packed, packed_fir_one_pol_fft, one_pol and generic; on the split and fused paths,
 * whose FIR has no separate output, it runs the one-pol FIR kernel instead. */
int fengine_debug_fir(fengine_t *fe, const void *in, float *g_out, int64_t n_spectra, void *stream);

/* Tuning knobs (optional; defaults are chosen at create).  key: "chunk_spectra" (spectra per
 * L2-resident chunk; 0 = whole call), "fir_rows" (spectra per FIR tile), "profile" (0/1, see below), "force_generic" (0/1: use the simple
 * one-thread-per-output kernels), "pol_packed" (0/1, default 1: allow the kernels that process both pols of an
 * antenna in packed FP32 lanes; they are used when n_pols = 2, n <= 8192 and the two pols of every antenna have
 * equal coarse delays), "fused" (0/1, default 0: run the pol-packed path as ONE persistent, warp-specialised kernel
 * whose FIR -> FFT transposition goes through an L2-resident ring of rows instead of a full-size HBM scratch,
 * fe_pipe.cuh; T = 2, 4, 8, 16; knobs "ring_rows", "fir_warps", "tracks", "segments", "pipe_ctas"), "split" (-1 / 0 / 1,
 * n = 4096, 16384, 32768, equal coarse delays in both pols: the first radix-16 stage of the transform runs in the FIR
 * kernel and the rest as independent n/16-point transforms, fe_split.cuh, the arrangement PAPER.md:403-409 proposes;
 * -1 (default) = where it measures faster, i.e. n >= 16384, 0 = never, 1 = wherever it exists), "fft_persistent" (0/1, default 0: the
 * pol-packed FFT as one persistent CTA per SM whose rows arrive by bulk copy into the exchange buffer, n <= 4096),
 * "scratch_fp16" (0/1, default 0; T = 16, n = 1024 or 4096, pol-packed path: the FIR output / FFT input is stored in
 * FP16 with FP32 arithmetic on both sides, the variant PAPER.md:407 proposes; NOT within the 1e-4 parity bar, it is
 * the comparison arm of the precision experiment of PAPER.md:149-157), "l2_persist" (bytes of L2 set aside for
 * persisting lines over the scratch of a chunked call, 0 = off), "host_chunks" (pieces of the fengine_process_host pipeline, 1 = no overlap),
 * "sample_bits" (4, 8, 10 (default), 12, 16: width of the packed input samples, same big-endian bit stream, sample u
 * in bits [b u, b u + b); the stream is then L*b/8 bytes.  The paper's bit-depth sweep.  Widths other
 * than 10 run the tiled kernels on the pol-packed path with 16 taps, else the generic kernels).  Returns INVALID_ARG for
 * unknown keys, and STATE for the options that change the data layout or the path ("sample_bits", "force_generic",
 * "pol_packed", "fused", "split", "scratch_fp16") while a stream is open. */
int fengine_set_option(fengine_t *fe, const char *key, int64_t value);

/*
 * Per-kernel timing for the roofline report.  With option "profile" = 1 every fengine_process call
 * records CUDA events on the caller's stream around each kernel.  fengine_profile_read waits for
 * them, returns the summed device time of the FIR kernel launches and of the FFT kernel launches
 * (milliseconds) and the number of launches of each since the last read, and clears the record.
 * fir_ms, fft_ms, n_fir, n_fft: HOST out-pointers (any may be NULL).
 */
int fengine_profile_read(fengine_t *fe, double *fir_ms, double *fft_ms, int64_t *n_fir, int64_t *n_fft);

/* Number of kernel launches the last fengine_process / _f32 call enqueued (for bench accounting). */
int64_t fengine_last_launch_count(const fengine_t *fe);

/* Test hook: with option "pipe_stats" = 1 the pipelined kernel accumulates 16 SM-clock counters per CTA (waits of its
 * three roles, rows per team; layout in csrc/fe_pipe.cuh).  Copies up to max_words of them to HOST `out`
 * ([n_sms][16] uint64) and zeroes them.  Synchronises the device. */
int fengine_debug_pipe_stats(fengine_t *fe, uint64_t *out, int64_t max_words);

/* Which kernels fengine_process would launch now (options, shape, equal or unequal coarse delays of the two pols):
 * a test hook, so that a parity test of a shape can assert that it exercised the tiled kernels it was written for
 * (every path computes steps 1-7 of PAPER.md:31-43).  Returns a FENGINE_PATH_* value, -1 for a null handle. */
enum {
    FENGINE_PATH_GENERIC = 0,                 /* one thread per output (any shape; slow, for tests) */
    FENGINE_PATH_ONE_POL = 1,                 /* fe_fir.cuh + fe_fft.cuh */
    FENGINE_PATH_POL_PACKED = 2,              /* fe_fir2.cuh / fe_fir3.cuh + fe_fft2.cuh */
    FENGINE_PATH_PACKED_FIR_ONE_POL_FFT = 3,  /* fe_fir2.cuh / fe_fir3.cuh + fe_fft.cuh (n >= 16384: 32 taps, other sample widths) */
    FENGINE_PATH_FUSED = 4,                   /* fe_pipe.cuh */
    FENGINE_PATH_SPLIT = 5                    /* fe_split.cuh */
};
int fengine_debug_path(const fengine_t *fe);

/* Measurement hook for the "alu" roofline (BASELINE.json north_star: "the FIR+FFT flops at FP32 peak"; the FIR of
 * Eq. (1), is 2T flops per sample in exactly this instruction form): runs a loop of packed FP32
 * multiply-adds (FFMA2, the FIR kernels' operand pattern) on every SM of the current device, a few launches timed with
 * CUDA events on the legacy stream, and writes the sustained rate in lane-operations (one FMA = one lane-operation)
 * per second to HOST *lane_ops_per_second and the time of one launch in ms to HOST *ms_per_launch (may be NULL).
 * Needs no handle; synchronises the device. */
int fengine_debug_fp32_rate(double *lane_ops_per_second, double *ms_per_launch);

#ifdef __cplusplus
}
#endif
#endif /* FENGINE_H */

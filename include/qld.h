/*
 * qld.h -- C ABI of the B200-native quadrature lock-in discrimination (QLD) hot path.
 *
 * Method: arXiv 1511.03390, "Real-time quadrature lock-in discrimination imaging through
 * scattering media".  Citations "P:<n>" are line numbers of the paper text;
 * "G<n>" are the readings listed in DESIGN.md section 2.
 *
 * For every pixel p of a stack of camera frames x_s(p), s = 1..N, and every reference k:
 *
 *     I_k(p) = sum_s x_s(p) * sin(theta_{k,s})     in-phase sum      (G1, G5)
 *     Q_k(p) = sum_s x_s(p) * cos(theta_{k,s})     quadrature sum
 *     theta_{k,s} = 2*pi*nu_k*s + phase_k          nu = f_mod / f_s   (G4, G7, G8)
 *     amplitude R_k(p) = sqrt(I_k^2 + Q_k^2)       (G2)         phase_k(p) = atan2(Q_k, I_k) (G6)
 *
 * No normalisation and no background removal unless asked for (G3, G9).
 *
 * General rules
 *  - Every function returns a qld_status (QLD_OK = 0, errors negative) unless stated otherwise; nothing
 *    aborts, throws or prints.  qld_last_error() gives a text for the last failure of a context.
 *  - All work is enqueued on CUDA streams; nothing blocks the host except qld_sync(), qld_push_done(block=1),
 *    qld_create(), qld_destroy() and the qld_read_* calls that say so.
 *  - "host" pointers are CPU memory (pinned for truly asynchronous copies; pageable works but serialises);
 *    "device" pointers are CUDA global memory of the current device.  The library never frees caller memory.
 *  - Frames are frame-major: frame f of a batch starts at byte f*H*W*bytes_per_sample, rows of W samples,
 *    no padding.  Maps are row-major [K][H][W] float32.
 *  - One context is not thread-safe; distinct contexts are independent.
 *  - There is no CPU fallback: without a CUDA device qld_create() fails with QLD_E_CUDA.
 */
#ifndef QLD_H
#define QLD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qld_ctx qld_ctx; /* opaque; one per stream of frames */

/* Sample formats.  QLD_U16 is a little-endian uint16 array.  QLD_U16_BE is the camera's raw 16-bit stream as it arrives over
 * a Camera-Link style interface with the most significant byte first ("a stream of 16-bit binary data (2-bytes)"
 * "stitch pairs of bytes and store values in an array of the appropriate data type"): the pairs are stitched inside the
 * kernels' loads (a byte-permute selector on the CUDA cores, the roles of the two accumulator rows on the tensor cores), so
 * the paper's thread T2 and its extra pass over the data do not exist.  Frames keep their size: 2 bytes per sample. */
typedef enum { QLD_U8 = 0, QLD_U16 = 1, QLD_U16_BE = 2 } qld_dtype;

typedef enum {
    QLD_OK = 0,
    QLD_E_INVAL = -1,       /* bad argument (sizes < 1, nu outside (0, 0.5), hop outside 1..N, null pointer ...) */
    QLD_E_NOMEM = -2,       /* device/host allocation failed, or caller workspace too small / misaligned */
    QLD_E_CUDA = -3,        /* a CUDA call failed; sticky; text in qld_last_error() */
    QLD_E_STATE = -4,       /* call not valid now: demod before N frames are stored, SLIDE before hop new frames */
    QLD_E_OVERRUN = -5,     /* push would overwrite frames a pending window still needs / store is full */
    QLD_E_UNSUPPORTED = -6  /* requested accumulation cannot be exact or safe for this (dtype, N, nu) */
} qld_status;

/* Accumulation (G11).
 *  FP32     : fp32 references (fp64 sincospi of the exactly reduced angle, rounded once), fp32 FMA on
 *             pedestal-subtracted samples (x - x_first(p), exact), pedestal term and finalise in fp64.
 *             Parity: <= 1e-5 relative (floored at the map median).
 *  INT_BINS : every reference must be rational (den > 0).  Phase-bin sums B_r = sum_{s: num*s mod den = r} x_s
 *             in int32, exact; I, Q = sum_r B_r * sin/cos(2*pi*r/den + phase) in fp64.  For den = 4 and a
 *             phase that is a multiple of pi/2 the references are integers {0, +-1} and I, Q are exact
 *             integers ("integer-valued reference" path).  QLD_E_UNSUPPORTED if a bin could overflow int32.
 *  INT_REFS : INT_BINS with the most compact exact form where one exists: for den = 3 or 6 and no phase offset the scaled
 *             references (2/sqrt3) sin theta_s in {0, +-1} and 2 cos theta_s in {+-1, +-2} are integers, so TWO exact int32 sums
 *             per reference suffice (2Q = 2B0+B1-B2-2B3-B4+B5, (2/sqrt3) I = B1+B2-B4-B5) instead of three bin
 *             rows: I = (sqrt3/2) row 0, Q = row 1 / 2.  Other references of the context keep their bin rows.  A third less
 *             accumulator traffic in a sliding update.  qld_get_bins then returns those two integer-reference sums.  A row of
 *             the compact form collects up to 4N/3 sample values (a bin row N/den): where max_value * (4N/3 + 2) reaches 2^31 the
 *             references keep their bin rows, and qld_accum_mode reports INT_BINS when none is compact.
 *  FIXED    : fixed-point references R(s) = rint(2^30 * sin/cos(theta_s)) (Q1.30 integers; the table can also
 *             be supplied, qld_set_ref_table_fixed).  I*2^30 = sum_s x_s R_sin(s), Q likewise, exact in int64:
 *             computed on the tcgen05 tensor cores as a [pixel bytes x frames].[frames x reference digits]
 *             int8 contraction (A6).  Bit-exact against an integer oracle with the same
 *             table; |R*2^-30 - sin| <= 2^-31, so the maps also agree with the float definition to ~1e-9.
 *             Whole-window stores (ring_frames 0 or -1): H*W*bytes a multiple of 16, N <= 65536.
 *             Rings (ring_frames > N, at most 2 references): the same exact sums, kept as int64 across hops by the
 *             bulk-copy sliding kernel (64-bit integer multiply-add on the CUDA cores) -- the sliding window of P:181-183
 *             with float references and no drift at all, at any nu; the table entry of a frame is a function of its
 *             absolute index and is extended per push.
 *  AUTO     : INT_REFS (= INT_BINS, compact where possible) when every reference is rational with den <= 16 and the bound holds; else FIXED for
 *             K >= 2 references on a whole-window store that meets FIXED's conditions (the CUDA-core kernel is
 *             instruction-bound there, the contraction is HBM-bound and more accurate than fp32); else FP32. */
typedef enum { QLD_ACC_AUTO = 0, QLD_ACC_FP32 = 1, QLD_ACC_INT_BINS = 2, QLD_ACC_FIXED = 3, QLD_ACC_INT_REFS = 4 } qld_accum;

typedef enum { QLD_NORM_PAPER = 0 /* no scaling (G3) */, QLD_NORM_AMPLITUDE = 1 /* I, Q, R times 2/N */ } qld_norm;

typedef enum { QLD_WHOLE = 0, QLD_SLIDE = 1 } qld_mode;

/* Which maps qld_demod produces (bit mask; unrequested maps are not computed or written). */
enum { QLD_MAP_I = 1, QLD_MAP_Q = 2, QLD_MAP_AMP = 4, QLD_MAP_PHASE = 8, QLD_MAP_ALL = 15,
       QLD_MAP_SUMS_I64 = 16 /* FIXED only: also keep the exact int64 sums, see qld_get_sums_i64 */ };

typedef struct {
    double nu;             /* f_mod/f_s in cycles per sample, 0 < nu < 0.5 (G18); ignored when den > 0 */
    double phase;          /* reference phase in radians (G7) */
    int64_t num, den;      /* den > 0: nu == num/den exactly, 0 < num/den < 1/2, angles reduced in integers */
    int32_t phase_quarter; /* adds phase_quarter * pi/2 exactly */
    int32_t reserved;
} qld_ref;

typedef struct {
    int32_t H, W;            /* frame size in pixels, >= 1 */
    int32_t dtype;           /* qld_dtype */
    int32_t N;               /* window length in frames, >= 1 */
    int32_t K;               /* number of references, 1..8 */
    const qld_ref *refs;     /* K entries, copied by qld_create */
    int32_t ring_frames;     /* 0: whole-window store of exactly N frames.  > 0: ring buffer for streaming,
                                must be > N; a producer pushing batches of b frames and a consumer sliding by hop
                                never stall each other when ring_frames >= N + hop + b - 1.
                                -1: no store: frames are attached with qld_attach_frames_device */
    int32_t accum;           /* qld_accum */
    int32_t norm;            /* qld_norm */
    int32_t maps;            /* mask of QLD_MAP_*; 0 means QLD_MAP_ALL */
    uint32_t max_value;      /* largest sample value the caller guarantees (0 = type maximum); used only for
                                the INT_BINS overflow bound */
    int32_t resync_hops;     /* SLIDE, FP32: recompute the window from the ring every this many hops, which bounds the drift of the
                                add/subtract update; 0 = automatic (every 16*ceil(N/hop) hops), < 0 = never */
    int32_t external_store;  /* 1: the frame store (N frames, or ring_frames frames) is the caller's device buffer, given
                                with qld_attach_frames_device; frames arrive in place and are announced with
                                qld_commit_frames (zero-copy ingest).  ring_frames = -1 implies it. */
    int32_t slide_hop;       /* > 0 (ring contexts): block-partial sliding (P:181-183 with a constant hop): the context keeps
                                the N/slide_hop per-batch partial sums of the window (N/slide_hop x rows x H*W accumulators)
                                and a QLD_SLIDE update reads only the slide_hop NEW frames: the expired batch's partial is
                                taken off instead of re-reading its frames.  Needs N % slide_hop == 0, every
                                qld_demod(QLD_SLIDE, hop) with hop == slide_hop, and frames the TMA kernel accepts
                                (H*W*bytes a multiple of 16, at least one 2 KB segment per SM, slide_hop >= 16..64
                                depending on the frame size): QLD_E_UNSUPPORTED otherwise.  Results are identical to the
                                frame re-reading update (bit-exact for INT_BINS). */
    int32_t window_relative; /* ring contexts: 1 = the I, Q and phase maps of a window that starts after a frames are turned back by
                                2 pi nu a, i.e. they are what references counted from the window's own first frame (s = 1)
                                would give: successive windows of a steady source then show a steady phase (reading G10,
                                P:181-183).  0 (default): references by absolute frame index.  The amplitude is the same either
                                way; qld_get_bins / qld_get_sums_i64 always hold absolute-index sums. */
    int32_t reserved2;
    int32_t ref_tables_supplied; /* 1: the caller supplies every reference table with qld_set_ref_tables before the first
                                qld_demod (QLD_E_STATE otherwise); refs[k].nu / num / den are then not used and not validated, so
                                nu = 0 and nu = 1/2 (reading G18) can be expressed.  FP32 / FIXED (or AUTO) on whole-window stores. */
    void *workspace;         /* device memory of qld_workspace_bytes() bytes, 256-byte aligned, owned by the
                                caller (e.g. a torch tensor) and kept alive until qld_destroy; NULL: the
                                library allocates and frees it */
    size_t workspace_bytes;
    void *compute_stream;    /* cudaStream_t for kernels (e.g. torch's current stream); NULL: library creates one */
    void *copy_stream;       /* cudaStream_t for host->device copies; NULL: library creates one */
} qld_config;

/* Size of the device workspace a context with this configuration needs (frame store or ring, reference
 * tables, accumulators, maps).  QLD_E_INVAL / QLD_E_UNSUPPORTED as for qld_create. */
int qld_workspace_bytes(const qld_config *cfg, size_t *bytes_out);

/* Build a context: validate, carve the workspace, fill the reference tables on the device (A1; P:99,
 * P:156 "creates tables of sine and cosine functions").  *ctx_out is NULL on failure. */
int qld_create(const qld_config *cfg, qld_ctx **ctx_out);

/* A2 ("thread T3 fetches data (raw frames)"): enqueue the copy of n_frames frames, host -> device
 * frame store, on the copy stream, and return.  The frames get absolute indices pushed+1 .. pushed+n.
 * The host buffer must stay unchanged until qld_push_done() reports completion.
 * Whole-window store: QLD_E_OVERRUN once N frames are stored (qld_reset starts the next stack).
 * Ring: QLD_E_OVERRUN if the push would overwrite a frame that a not-yet-requested window update needs;
 * QLD_E_INVAL if n_frames < 1 or n_frames > capacity. */
int qld_push_frames(qld_ctx *ctx, const void *host_frames, int n_frames);

/* Same, for frames that are already in device memory (device -> device copy on the copy stream). */
int qld_push_frames_device(qld_ctx *ctx, const void *device_frames, int n_frames);

/* Use the caller's device buffer in place (no copy).  The buffer must stay valid, and frames a pending demod
 * reads unchanged, while demods are in flight.
 * Whole-window store (ring_frames 0 / -1; with 0 the library's own store is left unused until qld_reset detaches the
 * buffer; qld_push_frames is refused with QLD_E_STATE while a buffer is attached): a buffer of N frames; counts as N
 * frames pushed.
 * Ring (ring_frames > 0, external_store = 1): a buffer of ring_frames frames; counts as no frames: announce
 * them with qld_commit_frames as they arrive. */
int qld_attach_frames_device(qld_ctx *ctx, const void *device_frames);

/* Zero-copy ingest (A2 for producers that write device memory themselves: a capture card doing peer-to-peer
 * DMA, a decode kernel, the synthetic filler).  external_store contexts only.  The caller has written -- or
 * has enqueued on `producer_stream` (cudaStream_t, NULL = already complete) the work that writes -- the next
 * n_frames frames, absolute indices pushed+1 .. pushed+n, in place: frame s lives at
 * store + ((s-1) mod capacity) * H*W*bytes_per_sample, capacity = ring_frames (ring) or N (whole store).
 * The call orders later demods after that work and extends the reference tables; it copies nothing.
 * Errors as qld_push_frames (QLD_E_OVERRUN: those slots still belong to a window that was not produced yet). */
int qld_commit_frames(qld_ctx *ctx, int n_frames, void *producer_stream);

/* Have all pushes issued so far completed (host buffers reusable)?  block = 0: returns QLD_OK when done,
 * QLD_E_STATE when still in flight.  block = 1: waits, then QLD_OK. */
int qld_push_done(qld_ctx *ctx, int block);

/* A3/A3'/A4/A5/A6 (P:99 Methods: the two sums and R(j,k); "the intensity at every pixel is multiplied by two
 * numbers ... accumulated", then "squared and added"; P:181-183 sliding sequence; P:49 several frequencies): enqueue one
 * demodulation on the compute stream; it waits (on the device) for every push
 * issued before it.
 *  QLD_WHOLE: the window is the most recent N frames stored (whole store: frames 1..N).  hop is ignored.
 *  QLD_SLIDE: ring contexts only.  The first call produces window 0 (frames 1..N); each later call advances
 *             the window by hop frames (1 <= hop <= N; window w = frames w*hop+1 .. w*hop+N for constant
 *             hop, G10), adding the hop new frames and subtracting the hop expired ones.
 * References are indexed by absolute frame number in both modes.
 * QLD_E_STATE if the frames the window needs are not all pushed yet.
 * Consecutive sliding updates may overlap on the device (the next launch ramps up while the previous one drains; it touches the
 * stored sums only once the previous launch is complete), so the maps of window w are defined for work ordered after THAT
 * qld_demod on the compute stream (qld_read_map, a kernel of the caller's on the same stream) or after qld_sync -- not for a
 * reader on an unrelated stream. */
int qld_demod(qld_ctx *ctx, int mode, int hop);

/* The processed images ("resulting in the 32-bit n x n processed image"; I and Q are the "two different 2-D arrays
 * that represent the two quadrature components"; amplitude per P:99; phase per reading G6).
 * Device pointers to the maps of reference k written by the last qld_demod: row-major [H][W] float32, valid
 * until the next qld_demod / qld_reset / qld_destroy; read them on the compute stream or after qld_sync().
 * Any out-pointer may be NULL.  A map that was not requested in cfg.maps comes back as NULL. */
int qld_get_maps(qld_ctx *ctx, int k, const float **I, const float **Q, const float **amp, const float **phase);

/* INT_BINS / INT_REFS only: device pointer to the exact int32 accumulators of reference k, [n_rows][H][W].  For even
 * den the rows are the differences D_r = B_r - B_{r+den/2}, r = 0..den/2-1 (n_rows = den/2); for odd den the
 * bins B_r (n_rows = den).  For den = 4, phase 0: D_0 = Q, D_1 = I exactly. */
int qld_get_bins(qld_ctx *ctx, int k, const int32_t **rows, int *n_rows);

/* Enqueue an asynchronous copy of one map of reference k (which = one QLD_MAP_* bit) to host memory on the
 * compute stream, after the last demod.  Complete after qld_sync(). */
int qld_read_map(qld_ctx *ctx, int k, int which, float *host_dst);

/* The reference table the kernels use: sin and cos of theta_{k,s} for s = s_first .. s_first+n-1, as float32
 * (FP32 accumulation) -- for inspection and tests.  Blocks until done.  Host pointers. */
int qld_read_ref_table(qld_ctx *ctx, int k, int64_t s_first, int n, float *sin_out, float *cos_out);

/* Caller-supplied reference tables (the main thread "creates tables of sine and cosine functions, appropriate for
 * the choice of lock-in and sampling frequencies"; "read from pre-calculated arrays"): replace the table of reference
 * k by sin_tab / cos_tab (host arrays of len == N doubles, entry i belongs to frame i+1, each in [-1, 1]).  The kernels
 * then compute I = sum_s x_s sin_tab[s-1], Q = sum_s x_s cos_tab[s-1] whatever the arrays hold.  FP32: each entry is
 * rounded once to float32; FIXED: to rint(2^30 * entry).  Whole-window stores only (QLD_E_UNSUPPORTED on rings and on
 * INT_BINS contexts).  Blocks until the device tables are rebuilt. */
int qld_set_ref_tables(qld_ctx *ctx, int k, const double *sin_tab, const double *cos_tab, int64_t len);

/* QLD_ACC_FIXED only.  Replace the Q1.30 reference table of reference k by caller-supplied integers (host arrays, each
 * entry in [-2^30, 2^30]); blocks until the device table is rebuilt.  Whole-window store: n == N entries, entry i belongs to
 * frame i+1.  Ring: the entries of the n most recently pushed frames (1 <= n <= frames pushed), to be called after the push
 * that brought them and before the qld_demod that uses them.  qld_read_ref_table_fixed copies the table in use back to the
 * host (blocks). */
int qld_set_ref_table_fixed(qld_ctx *ctx, int k, const int32_t *sin_q30, const int32_t *cos_q30, int n);
/* N entries each.  Whole-window store: frames 1..N.  Ring: the N most recently pushed frames. */
int qld_read_ref_table_fixed(qld_ctx *ctx, int k, int32_t *sin_q30, int32_t *cos_q30);

/* QLD_ACC_FIXED with QLD_MAP_SUMS_I64 (whole-window stores) or QLD_ACC_FIXED on a ring (always available: the sums the
 * context keeps across hops): device pointers to the exact sums sum_s x_s R(s) of reference k over the current window,
 * [H][W] int64 each (I*2^30 and Q*2^30 before normalisation), valid like the maps. */
int qld_get_sums_i64(qld_ctx *ctx, int k, const int64_t **I, const int64_t **Q);

/* Bookkeeping (host side, never blocks): frames pushed so far, windows produced so far. */
int qld_counters(const qld_ctx *ctx, int64_t *frames_pushed, int64_t *windows_done);

/* Life cycle.  The paper's threads hand frames and images over with status flags ("a flag indicates the
 * status"); here that hand-over is stream order, and these three are the only host-side waits:
 *  qld_sync    waits for both streams (all pushes copied, all demods finished: maps and host copies are valid);
 *  qld_reset   forgets all frames and accumulators -- the next push is frame 1 (t_1) of a new acquisition; a buffer
 *              attached in place of a whole-window store is detached, an attached ring stays attached;
 *  qld_destroy waits for pending work and frees what the library allocated; NULL is a no-op. */
int qld_sync(qld_ctx *ctx);
int qld_reset(qld_ctx *ctx);
void qld_destroy(qld_ctx *ctx);

/* Text of the last error of this context ("" if none).  ctx may be NULL: text of the last failed qld_create
 * on this thread. */
const char *qld_last_error(const qld_ctx *ctx);

/* Launch statistics for benchmarks: kernels launched by this context so far. */
int64_t qld_kernel_launches(const qld_ctx *ctx);

/* Introspection for benchmarks and tests: the accumulation mode in use (a qld_accum other than AUTO; negative
 * status if ctx is NULL), and the name of the kernel the last qld_demod launched ("" before the first):
 * "k_demod_stream", "k_demod_whole", "k_demod_tc", "k_slide_bulk" or "k_demod_slide".  Never NULL. */
int qld_accum_mode(const qld_ctx *ctx);
const char *qld_last_kernel(const qld_ctx *ctx);

/* Debug / test hook: force the tile shape of the next launches of this context instead of the automatic choice (an
 * invalid shape is ignored).  which = 0: k_demod_stream, a = SEG (contiguous bytes of every frame per tile, a power of two
 * <= 2048), b = KC (frames per pipeline stage); forcing also lifts the frame-size threshold, so small frames go through
 * the TMA-fed kernel.  which = 1: k_demod_tc, a = T (128-byte spans per tile), b = STAGES, c = KC (32 or 64).
 * which = 2: the sliding update: a = 1 always runs k_slide_bulk (also on frames too small to give every SM a tile), a = 2
 * never, a = 0 automatic.  For which = 0 / 1, a = 0 restores the automatic choice.  Results never depend on the shape (tests/ run every shape against the oracle). */
int qld_debug_set_tile(qld_ctx *ctx, int which, int a, int b, int c);

/* Contrast-to-noise ratio of a processed image (Eq. (1), Fig. 6; the paper's quality metric, the step
 * after the path):  CNR = (mean_s - mean_surr) / sqrt( mean over the slice of (I(j,k) - mean_surr)^2 ), mean_s
 * over the m x m source square with top-left pixel (y0, x0), the slice being the m-pixel wide square ring around
 * it (8 m^2 pixels, which must lie inside the frame: QLD_E_INVAL otherwise).  map_device: row-major [H][W] float32
 * in device memory (e.g. an amplitude map from qld_get_maps).  Enqueued on `stream` (cudaStream_t or NULL); writes
 * out_device[0..3] = {CNR, mean_s, mean_surr, rms} (device memory, 4 doubles); fp64 arithmetic, IEEE inf / nan when
 * the slice is flat. */
int qld_cnr(const float *map_device, int32_t H, int32_t W, int32_t y0, int32_t x0, int32_t m, double *out_device, void *stream);

/* Unknown-frequency search ("a series of QLDs ... at different frequencies"; P:99 the FFT image |F(j,k,omega_q)|^2;
 * SURVEY.md 8(f2)): demodulate the N-frame stack `frames_device` (frame-major, device memory, qld_dtype) at every DFT
 * bin q = q_lo..q_hi (nu = q/N, 1 <= q_lo <= q_hi, 2*q_hi < N) and keep, per pixel, the largest amplitude R_q = |F_q|
 * and its bin (the lowest bin on a tie): amp_max_device [H][W] float32, bin_device [H][W] int32 (device memory).
 * Frames whose byte size is a multiple of 16: 32 bins per pass over the stack, one tcgen05 launch per pass (Q1.30 references,
 * exact sums, arg-max fused into the epilogue), N/64 passes in all.  Other frame sizes: eight bins per pass through a context
 * (FP32).  Work is enqueued on `stream` (cudaStream_t; NULL = the legacy default stream); the call returns after
 * the last pass has finished. */
int qld_dominant_bin(const void *frames_device, int32_t dtype, int32_t H, int32_t W, int32_t N, int32_t q_lo, int32_t q_hi,
                     float *amp_max_device, int32_t *bin_device, void *stream);

/* qld_dominant_bin for callers that cannot allocate device memory -- a camera loop that must not stall on the driver lock
 * cudaMalloc / cudaFree take (the real-time threads), or a process whose HBM another allocator already holds in
 * full.  Same search, same arguments, same results as the tensor-core route of qld_dominant_bin, but its scratch
 * (the Q1.30 digit tiles of the bins, two tile counters) lives in one fixed array inside the library instead of pool memory;
 * the call issues no cudaMalloc, cudaFree or other allocating routine.  The caller still owns and passes the inputs and outputs.
 *   Limits: the digit tiles take 256 * (N rounded up to a multiple of 128) * ceil((q_hi - q_lo + 1) / 32) bytes (qld_dominant_bin_static_bytes
 * computes it) and must fit QLD_SEARCH_STATIC_BYTES = 4 MiB -- e.g. all 511 bins of an N = 1024 window, or 128 bins of N = 4096;
 * a larger search returns QLD_E_NOMEM (split the bin range over several calls and combine, or use qld_dominant_bin).  Only frames
 * whose byte size is a multiple of 16 in a 16-byte aligned stack: QLD_E_UNSUPPORTED otherwise (the other route builds contexts).
 * Every GPU on which this library's kernels are loaded holds the array (4 MiB + 256 B) until the process exits.
 *   First call on a device: looks up the array's address on that device (the device must be current, as for every call
 * here) and, if nothing ran from the library on it before, loads the kernels; make that call during set-up, before any
 * stream capture begins.  Later calls on the device do no set-up.
 *   Sharing: all calls on one device use the same array, which keeps the last call's contents; the entry point re-zeroes
 * the counters and rewrites every digit it reads, so calls one after the other are independent.  Two calls whose GPU work
 * overlaps (two host threads, two streams) race on it and give wrong maps: serialise them.  The call returns after the last
 * pass has finished (it synchronises `stream` only).
 *   Errors: QLD_E_INVAL as qld_dominant_bin, QLD_E_NOMEM / QLD_E_UNSUPPORTED as above, QLD_E_CUDA; the text of this thread's
 * last failure is at qld_dominant_bin_static_error() ("" after a success; never NULL). */
#define QLD_SEARCH_STATIC_BYTES (4 << 20)
int qld_dominant_bin_static(const void *frames_device, int32_t dtype, int32_t H, int32_t W, int32_t N, int32_t q_lo, int32_t q_hi,
                            float *amp_max_device, int32_t *bin_device, void *stream);
int64_t qld_dominant_bin_static_bytes(int32_t N, int32_t q_lo, int32_t q_hi);   /* scratch bytes of that search; QLD_E_INVAL (< 0) for a bad range */
const char *qld_dominant_bin_static_error(void);

/* Measuring stick for the benchmark, not a step of the path (the read-only ceiling; P:181 is why reads are
 * what matters -- QLD keeps two n^2 arrays beside the frames): loads every 16-byte word of buf_device[0 .. bytes) once (bytes
 * rounded down to a multiple of 16; the buffer 16-byte aligned, in device memory) and writes one checksum word per CTA to
 * out_device (QLD_PROBE_OUT_WORDS uint32 of device memory; word b = the sum over CTA b's words of x ^ y ^ z ^ w of each 16-byte
 * load, mod 2^32).  One launch enqueued on `stream` (cudaStream_t or NULL); time it with events around the call: bytes / time is
 * the read bandwidth this GPU sustains, the ceiling bench.py quotes beside the copy peak. */
#define QLD_PROBE_OUT_WORDS 4096
int qld_probe_read(const void *buf_device, int64_t bytes, uint32_t *out_device, void *stream);

/* Display mapping (the processed 32-bit image "is displayed on the computer monitor"; there is no graphics stack
 * here, the 8-bit image is delivered to device memory; reading G22): lo / hi = smallest / largest non-NaN value
 * of the n floats at map_device, out_device[i] = rint(255 * (x_i - lo) / (hi - lo)) clamped to 0..255 (0 for NaN and
 * for a flat map).  range_device (2 floats, may be NULL) receives {lo, hi}; scratch_device: 8 bytes of device memory.
 * Three small launches enqueued on `stream` (cudaStream_t or NULL). */
int qld_display_map(const float *map_device, int64_t n, uint8_t *out_device, float *range_device, void *scratch_device, void *stream);

/* ---- synthetic input filler (not part of the method; device twin of paper_1511_03390_b200/synth.py) ---- */
typedef struct {
    int32_t H, W;
    int32_t dtype;            /* qld_dtype */
    uint32_t maxval;
    uint64_t key;             /* noise-stream key (synth.seed_key(seed, 1)) */
    int32_t n_terms;          /* J: number of weight maps / modulation rows, 0..8 */
    int32_t has_disk;
    const float *base;        /* device, [H*W] */
    const float *weights;     /* device, [J][H*W] */
    const double *mods;       /* device, [J][mod_stride], indexed by absolute frame s */
    int64_t mod_stride;
    double noise_a, noise_b;
    int32_t disk_x0, disk_cy, disk_radius, reserved;
    double disk_amp;
    const double *disk_mod;   /* device, indexed by absolute frame s */
} qld_synth_scene;

/* Fill n_frames frames s_first .. s_first+n-1 into device memory `out` (frame-major) on `stream`
 * (cudaStream_t or NULL).  Bit-identical to synth.frames(). */
int qld_synth_fill(const qld_synth_scene *scene, int64_t s_first, int n_frames, void *out_device, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* QLD_H */

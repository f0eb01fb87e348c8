// C-ABI entry points of libqld.so (include/qld.h): context, frame ingest (A2), stream/event ordering, and the
// host-side bookkeeping of whole-window and sliding-window demodulation.  No arithmetic of the method runs on
// the host: reference tables, bin combine weights, sums and maps are all produced by the kernels in qld_tables.cu,
// qld_kernels.cu, qld_stream.cu and qld_tc.cu; the host only plans buffers, orders streams and keeps counters.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <new>
#include <string>

#include <nvtx3/nvToolsExt.h>

#include "qld_internal.h"
#include "qld_slide.h"
#include "qld_stream.h"
#include "qld_tc.h"

namespace {

constexpr int N_PUSH_EVENTS = 64;
constexpr int N_DEMOD_EVENTS = 32;

thread_local std::string g_create_error;

// NVTX range around a host-side entry point (push / demod / read): shows up in Nsight timelines, costs nothing without a tool
struct NvtxRange {
    explicit NvtxRange(const char *name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};

struct DemodEvent {
    cudaEvent_t ev;
    int64_t oldest_read;   // oldest absolute frame index the demod reads
    bool used;
};

}  // namespace

struct qld_ctx {
    // configuration
    int H, W, dtype, bytes, N, K, accum, norm, maps, resync_hops;
    int big_endian;          // QLD_U16_BE: byte pairs stitched most significant byte first
    int window_relative;     // cfg.window_relative: I / Q / phase maps turned back to window-relative references
    int64_t HW;
    uint32_t max_value;
    int cap, cap_w;          // frame store capacity, weight table capacity
    bool ring, external;     // ring buffer / frames attached by the caller
    bool is_int, is_fixed;
    bool fix_ring;           // FIXED on a ring: Q1.30 references, int64 sums kept across hops by k_slide_bulk
    bool tc_bins;            // integer bins may run as a one-digit int8 contraction on the tensor cores (digits = bin indicators)
    int rows, rows_pad;
    RefPlan ref[QLD_MAX_K];
    FinParams fin;
    // tensor-core (FIXED) path
    int32_t *rfix;           // [2K][N] Q30 references
    int8_t *digits;          // digit tiles for the MMA B operand
    int64_t *sums;           // optional [2K][HW] exact sums
    unsigned int *tile_counter;   // three counters in rotation: each launch zeroes the next launch's one
    unsigned int counter_flip;
    alignas(64) unsigned char tmap[256];   // two CUtensorMap (qld_tc_encode_tmap)
    bool tmap_valid;
    int n_sms;
    // TMA-fed CUDA-core path (qld_stream.cu)
    alignas(64) unsigned char stream_tmap[128];
    const void *stream_tmap_frames;   // frame store the map was encoded for (NULL: none yet)
    StreamShape stream_shape;
    // bulk-copy sliding update (qld_slide.cu)
    alignas(64) unsigned char slide_tmap[128];
    const void *slide_tmap_frames;
    SlideShape slide_shape;
    int dbg_slide;           // qld_debug_set_tile(which = 2): 0 automatic, 1 always k_slide_bulk, 2 never
    // device memory
    void *ws;
    bool own_ws;
    size_t ws_bytes;
    unsigned char *frames;   // store (or attached buffer)
    unsigned char *own_frames; // the library-owned store (NULL on external contexts)
    int dbg_stream[2], dbg_tc[3]; // qld_debug_set_tile overrides (zeros: automatic)
    bool tables_supplied;    // cfg.ref_tables_supplied: tables come from qld_set_ref_tables
    unsigned tables_set;     // bit k: reference k has its table
    void *wtab;
    double *cum;
    void *acc;
    float *ped;
    unsigned char *part;     // block-partial sliding: [M][rows_pad][HW] partial sums (int32 / double)
    int slide_hop, n_part;   // hop of the partial mode (0: off), M = N / hop
    float *mapI, *mapQ, *mapA, *mapP;
    // streams and events
    cudaStream_t s_comp, s_copy;
    bool own_comp, own_copy;
    cudaEvent_t push_ev[N_PUSH_EVENTS];
    int push_ev_next;
    bool push_pending;
    uint64_t push_seq, waited_seq;   // push events recorded / the last one the compute stream was made to wait for
    int64_t tab_filled;      // ring: reference tables are filled up to this absolute frame index (they may run ahead of the frames)
    DemodEvent demod_ev[N_DEMOD_EVENTS];
    int demod_ev_next;
    cudaEvent_t tables_ev;
    // state
    int64_t pushed;          // frames pushed since reset (absolute index of the newest frame)
    int64_t windows_done;
    bool seeded;             // sliding accumulators valid
    int64_t win_start;       // 0-based offset a of the current window: frames a+1 .. a+N
    int64_t hops_since_seed;
    int64_t launches;
    const char *last_kernel;
    bool sticky;
    std::string err;
};

namespace {

int fail(qld_ctx *c, int code, const char *msg)
{
    if (c) c->err = msg; else g_create_error = msg;
    return code;
}

int cuda_fail(qld_ctx *c, cudaError_t e, const char *what)
{
    char buf[256];
    snprintf(buf, sizeof buf, "%s: %s", what, cudaGetErrorString(e));
    if (c) { c->err = buf; c->sticky = true; } else g_create_error = buf;
    return QLD_E_CUDA;
}

#define CU(c, call)                                              \
    do {                                                         \
        cudaError_t e_ = (call);                                 \
        if (e_ != cudaSuccess) return cuda_fail((c), e_, #call); \
    } while (0)

size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

int64_t gcd64(int64_t a, int64_t b) { while (b) { int64_t t = a % b; a = b; b = t; } return a; }

struct Plan {
    int H, W, dtype, bytes, N, K, accum, norm, maps, cap, cap_w, rows, rows_pad;
    bool ring, external, is_int, is_fixed, fix_ring;
    bool tc_bins;            // INT_BINS on a whole-window store whose shape the tensor-core contraction accepts
    int64_t HW;
    RefPlan ref[QLD_MAX_K];
    FinParams fin;
    // workspace offsets
    int slide_hop;
    size_t off_part;
    size_t off_frames, off_wtab, off_cum, off_acc, off_ped, off_I, off_Q, off_A, off_P, off_rfix, off_digits, off_sums, off_counter, total;
};

int make_plan(const qld_config *cfg, Plan *pl, std::string *err)
{
    auto bad = [&](int code, const char *m) { *err = m; return code; };
    if (!cfg) return bad(QLD_E_INVAL, "config is NULL");
    if (cfg->H < 1 || cfg->W < 1) return bad(QLD_E_INVAL, "H and W must be >= 1");
    if (cfg->dtype != QLD_U8 && cfg->dtype != QLD_U16 && cfg->dtype != QLD_U16_BE) return bad(QLD_E_INVAL, "dtype must be QLD_U8, QLD_U16 or QLD_U16_BE");
    if (cfg->N < 1) return bad(QLD_E_INVAL, "N must be >= 1");
    if (cfg->K < 1 || cfg->K > QLD_MAX_K || !cfg->refs) return bad(QLD_E_INVAL, "K must be 1..8 with refs given");
    if (cfg->ring_frames < -1 || (cfg->ring_frames > 0 && cfg->ring_frames <= cfg->N))
        return bad(QLD_E_INVAL, "ring_frames must be -1, 0, or > N");
    if (cfg->accum < QLD_ACC_AUTO || cfg->accum > QLD_ACC_INT_REFS) return bad(QLD_E_INVAL, "unknown accum");
    if (cfg->external_store != 0 && cfg->external_store != 1) return bad(QLD_E_INVAL, "external_store must be 0 or 1");
    if (cfg->slide_hop < 0 || cfg->slide_hop > cfg->N) return bad(QLD_E_INVAL, "slide_hop must be 0..N");
    if (cfg->slide_hop > 0 && cfg->ring_frames <= 0) return bad(QLD_E_INVAL, "slide_hop needs a ring context");
    if (cfg->norm != QLD_NORM_PAPER && cfg->norm != QLD_NORM_AMPLITUDE) return bad(QLD_E_INVAL, "unknown norm");
    if (cfg->maps & ~(QLD_MAP_ALL | QLD_MAP_SUMS_I64)) return bad(QLD_E_INVAL, "unknown bits in maps");
    if (cfg->window_relative != 0 && cfg->window_relative != 1) return bad(QLD_E_INVAL, "window_relative must be 0 or 1");
    if (cfg->ref_tables_supplied != 0 && cfg->ref_tables_supplied != 1) return bad(QLD_E_INVAL, "ref_tables_supplied must be 0 or 1");
    if (cfg->ref_tables_supplied && cfg->ring_frames > 0) return bad(QLD_E_UNSUPPORTED, "ref_tables_supplied: whole-window stores only");
    if (cfg->ref_tables_supplied && cfg->accum == QLD_ACC_INT_BINS) return bad(QLD_E_UNSUPPORTED, "ref_tables_supplied: FP32 or FIXED accumulation");
    memset(pl, 0, sizeof *pl);
    pl->H = cfg->H; pl->W = cfg->W; pl->dtype = cfg->dtype; pl->bytes = cfg->dtype == QLD_U8 ? 1 : 2;
    pl->N = cfg->N; pl->K = cfg->K; pl->norm = cfg->norm; pl->maps = (cfg->maps & QLD_MAP_ALL) ? cfg->maps : (cfg->maps | QLD_MAP_ALL);
    pl->HW = (int64_t)cfg->H * cfg->W;
    pl->ring = cfg->ring_frames > 0; pl->external = cfg->ring_frames == -1 || cfg->external_store == 1;
    pl->cap = pl->ring ? cfg->ring_frames : cfg->N;
    pl->cap_w = pl->cap + 1;

    bool all_rational = true;
    int64_t max_den = 0;
    for (int k = 0; k < cfg->K; ++k) {
        const qld_ref &r = cfg->refs[k];
        RefPlan &rp = pl->ref[k];
        rp.phase = r.phase; rp.phase_quarter = r.phase_quarter;
        if (!isfinite(r.phase)) return bad(QLD_E_INVAL, "phase must be finite");
        if (cfg->ref_tables_supplied) {                    // nu is whatever the caller's tables encode (G18)
            rp.nu = r.nu; rp.num = 0; rp.den = 0;
            all_rational = false;
        } else if (r.den > 0) {
            if (r.den >= (1ll << 31) || r.num <= 0 || 2 * r.num >= r.den) return bad(QLD_E_INVAL, "need 0 < num/den < 1/2 and den < 2^31");
            const int64_t g = gcd64(r.num, r.den);
            rp.num = r.num / g; rp.den = r.den / g; rp.nu = (double)rp.num / (double)rp.den;
            if (rp.den > max_den) max_den = rp.den;
        } else {
            if (!(r.nu > 0.0 && r.nu < 0.5)) return bad(QLD_E_INVAL, "nu must lie in (0, 0.5)");
            rp.nu = r.nu; rp.num = 0; rp.den = 0;
            all_rational = false;
        }
    }
    // accumulation mode
    const uint64_t vmax = cfg->max_value ? cfg->max_value : (cfg->dtype == QLD_U8 ? 255u : 65535u);
    // INT_REFS: references with den = 3 or 6 and no phase offset take the two-row integer-reference form
    // (their weights 2 cos theta_s run through +-2, +-1, +-1 per half period: at most 4N/3 + 2/3 sample values land in a row; a
    // reference whose two rows could overflow int32 keeps its plain bin rows, whose bound is N/den)
    const int64_t compact_per_row = (4 * (int64_t)cfg->N + 2) / 3 + 1;
    const bool compact_fits = (unsigned __int128)vmax * (uint64_t)(compact_per_row + 1) < (1ull << 31);
    auto compact = [&](int k, bool want) {
        const RefPlan &rp = pl->ref[k];
        return want && compact_fits && (rp.den == 3 || rp.den == 6) && rp.phase == 0.0 && (rp.phase_quarter & 3) == 0;
    };
    auto bins_rows = [&](int *rows_out, bool want_compact) {
        int rows = 0;
        for (int k = 0; k < cfg->K; ++k) {
            const int64_t den = pl->ref[k].den;
            rows += compact(k, want_compact) ? 2 : (int)((den % 2 == 0) ? den / 2 : den);
        }
        *rows_out = rows;
        return rows <= QLD_MAX_ROWS;
    };
    auto bins_fit = [&](bool want_compact) {   // |row sum| <= vmax * (number of frames that can land in one row)
        for (int k = 0; k < cfg->K; ++k) {
            const int64_t den = pl->ref[k].den;
            // a difference row takes +x from bin r and -x from bin r+den/2: magnitude bounded by one bin's sum; an
            // integer-reference row: see compact_per_row
            const int64_t per_row = compact(k, want_compact) ? compact_per_row : ((int64_t)cfg->N + den - 1) / den;
            if ((unsigned __int128)vmax * (uint64_t)(per_row + 1) >= (1ull << 31)) return false;
        }
        return true;
    };
    int acc = cfg->accum;
    int rows = 0;
    if (acc == QLD_ACC_AUTO) {
        // bins when the references allow them (exact, cheapest); for K >= 2 float references on a whole-window
        // store the CUDA-core kernel is instruction-issue bound (measured on the cfg2 stack: K = 2 5.8 TB/s, K = 3 3.6 TB/s
        // against 6.2-6.4 TB/s for the contraction) and the exact int8 contraction on the tensor
        // cores is used; otherwise (K = 1: the CUDA cores sit on the HBM roof) pedestal-subtracted fp32
        const bool tc_ok = !pl->ring && cfg->K >= 2 && (pl->HW * pl->bytes) % 16 == 0 && cfg->N <= 65536 && !(cfg->maps & ~(QLD_MAP_ALL | QLD_MAP_SUMS_I64));
        acc = (all_rational && max_den <= 16 && bins_rows(&rows, true) && bins_fit(true)) ? QLD_ACC_INT_REFS : (tc_ok ? QLD_ACC_FIXED : QLD_ACC_FP32);
    }
    const bool want_compact = acc == QLD_ACC_INT_REFS;
    if (acc == QLD_ACC_INT_BINS || acc == QLD_ACC_INT_REFS) {
        if (!all_rational) return bad(QLD_E_UNSUPPORTED, "INT_BINS needs every reference rational (den > 0)");
        if (!bins_rows(&rows, want_compact)) return bad(QLD_E_UNSUPPORTED, "INT_BINS: more than 16 bin rows in total");
        if (!bins_fit(want_compact)) return bad(QLD_E_UNSUPPORTED, "INT_BINS: a bin sum could overflow int32 for this N and max_value");
        if (want_compact) {                                  // no reference took the compact form: these are plain bins, say so
            bool any = false;
            for (int k = 0; k < cfg->K; ++k) any = any || compact(k, true);
            if (!any) acc = QLD_ACC_INT_BINS;
        }
    }
    if (acc == QLD_ACC_FIXED && pl->ring) {
        if (cfg->K > 2) return bad(QLD_E_UNSUPPORTED, "FIXED on a ring: at most 2 references");
        if ((pl->HW * pl->bytes) % 16 != 0) return bad(QLD_E_UNSUPPORTED, "FIXED: H*W*bytes_per_sample must be a multiple of 16");
        if ((int64_t)cfg->N > 65536) return bad(QLD_E_UNSUPPORTED, "FIXED: N must be <= 65536");
        const int nm = cfg->K * (((pl->maps & QLD_MAP_I) != 0) + ((pl->maps & QLD_MAP_Q) != 0) + ((pl->maps & QLD_MAP_AMP) != 0) + ((pl->maps & QLD_MAP_PHASE) != 0));
        if (qld_slide_shape(cfg->dtype, 2, cfg->K == 1 ? 2 : 4, cfg->slide_hop > 0, nm, pl->HW, reinterpret_cast<const void *>(16), 1, 1).seg == 0)
            return bad(QLD_E_UNSUPPORTED, "FIXED on a ring: the per-tile state (sums, partial sums, maps) does not fit shared memory: request fewer maps");
    } else if (acc == QLD_ACC_FIXED) {
        if ((pl->HW * pl->bytes) % 16 != 0) return bad(QLD_E_UNSUPPORTED, "FIXED: H*W*bytes_per_sample must be a multiple of 16 (TMA row pitch)");
        if ((int64_t)cfg->N > 65536) return bad(QLD_E_UNSUPPORTED, "FIXED: N must be <= 65536 for exact int32 partial sums");
    }
    if ((pl->maps & QLD_MAP_SUMS_I64) && acc != QLD_ACC_FIXED) return bad(QLD_E_INVAL, "QLD_MAP_SUMS_I64 needs QLD_ACC_FIXED");
    pl->accum = acc;
    pl->is_int = acc == QLD_ACC_INT_BINS || acc == QLD_ACC_INT_REFS;
    pl->is_fixed = acc == QLD_ACC_FIXED && !pl->ring;
    pl->fix_ring = acc == QLD_ACC_FIXED && pl->ring;
    FinParams &f = pl->fin;
    f.K = cfg->K; f.is_int = pl->is_int;
    f.scale = cfg->norm == QLD_NORM_AMPLITUDE ? 2.0 / (double)cfg->N : 1.0;
    if (pl->is_int) {
        int off = 0;
        for (int k = 0; k < cfg->K; ++k) {
            RefPlan &rp = pl->ref[k];
            rp.use_diff = compact(k, want_compact) ? 2 : (rp.den % 2 == 0 ? 1 : 0);
            rp.n_rows = rp.use_diff == 2 ? 2 : (int)(rp.use_diff ? rp.den / 2 : rp.den);
            rp.row_off = off;
            f.row_off[k] = off; f.n_rows[k] = rp.n_rows;
            off += rp.n_rows;                   // f.sw / f.cw are filled on the device by qld_create (k_bin_weights)
        }
        pl->rows = off;
    } else {
        for (int k = 0; k < cfg->K; ++k) {
            pl->ref[k].row_off = 2 * k; pl->ref[k].n_rows = 2;
            f.row_off[k] = 2 * k; f.n_rows[k] = 2;
        }
        pl->rows = 2 * cfg->K;
    }
    // kernel instantiations exist for 2, 3, 4, 8 and 16 rows (3: one reference with den = 6, e.g. BASELINE.json configs[3])
    pl->rows_pad = pl->rows <= 2 ? 2 : pl->rows <= 3 ? 3 : pl->rows <= 4 ? 4 : pl->rows <= 8 ? 8 : 16;

    // workspace layout
    size_t o = 0;
    pl->off_frames = o; if (!pl->external) o += align_up((size_t)pl->cap * pl->HW * pl->bytes);
    const bool cc = !pl->is_fixed;          // CUDA-core paths: weight tables, sliding accumulators, pedestal
    pl->off_wtab = o; if (cc) o += align_up((size_t)pl->cap_w * pl->rows_pad * 4);
    pl->off_cum = o; if (cc) o += align_up((size_t)pl->cap_w * pl->rows_pad * 8);
    pl->off_acc = o; if (cc && (pl->ring || pl->is_int)) o += align_up((size_t)pl->rows_pad * pl->HW * (pl->is_int ? 4 : 8));
    pl->off_ped = o; if (cc && pl->ring) o += align_up((size_t)pl->HW * 4);
    pl->slide_hop = cfg->slide_hop;
    pl->off_part = o;
    if (cfg->slide_hop > 0) {
        if (cfg->N % cfg->slide_hop != 0) return bad(QLD_E_UNSUPPORTED, "slide_hop must divide N");
        if ((pl->HW * pl->bytes) % 16 != 0) return bad(QLD_E_UNSUPPORTED, "slide_hop: H*W*bytes_per_sample must be a multiple of 16");
        o += align_up((size_t)(cfg->N / cfg->slide_hop) * pl->rows_pad * pl->HW * (pl->is_int ? 4 : 8));
    }
    const size_t map = align_up((size_t)pl->K * pl->HW * 4);
    pl->off_I = o; if (pl->maps & QLD_MAP_I) o += map;
    pl->off_Q = o; if (pl->maps & QLD_MAP_Q) o += map;
    pl->off_A = o; if (pl->maps & QLD_MAP_AMP) o += map;
    pl->off_P = o; if (pl->maps & QLD_MAP_PHASE) o += map;
    pl->off_rfix = o; if (pl->is_fixed) o += align_up((size_t)2 * pl->K * pl->N * 4);
    pl->off_digits = o;
    if (pl->is_fixed) o += align_up(qld_tc_digit_bytes(pl->K, pl->N));
    else if (pl->is_int && !pl->ring && (pl->HW * pl->bytes) % 16 == 0 && pl->N <= 65536) { pl->tc_bins = true; o += align_up(qld_tc_digit_bytes(2, pl->N)); }   // bins on the tensor cores
    pl->off_sums = o; if (pl->is_fixed && (pl->maps & QLD_MAP_SUMS_I64)) o += align_up((size_t)2 * pl->K * pl->HW * 8);
    pl->off_counter = o; o += 512;            // tile counter of the persistent kernels (+256: 32 doubles of scratch)
    pl->total = o;
    return QLD_OK;
}

int fill_tables(qld_ctx *c, int64_t s_first, int n, cudaStream_t st)
{
    TableFillParams tp;
    memset(&tp, 0, sizeof tp);
    tp.K = c->K; tp.is_int = c->is_int ? 1 : (c->fix_ring ? 2 : 0); tp.rows = c->rows_pad;
    for (int k = 0; k < c->K; ++k) tp.ref[k] = c->ref[k];
    tp.s_first = s_first; tp.n = n; tp.cap_w = c->cap_w; tp.wtab = c->wtab; tp.cum = c->cum;
    CU(c, qld_launch_table_fill(tp, st));
    c->launches++;
    return QLD_OK;
}

int init_device_state(qld_ctx *c)
{
    CU(c, cudaMemsetAsync(c->tile_counter, 0, 3 * sizeof(unsigned int), c->s_copy));
    // tables zeroed (padding rows stay zero; cum entry of frame 0 is zero), then filled for the whole store
    if (!c->is_fixed) {
        CU(c, cudaMemsetAsync(c->wtab, 0, (size_t)c->cap_w * c->rows_pad * 4, c->s_copy));
        CU(c, cudaMemsetAsync(c->cum, 0, (size_t)c->cap_w * c->rows_pad * 8, c->s_copy));
    }
    if (c->tables_supplied) {
        if (c->is_fixed) CU(c, cudaMemsetAsync(c->rfix, 0, (size_t)2 * c->K * c->N * 4, c->s_copy));
    } else if (c->is_fixed) {
        TableFillParams tp;
        memset(&tp, 0, sizeof tp);
        tp.K = c->K;
        for (int k = 0; k < c->K; ++k) tp.ref[k] = c->ref[k];
        tp.s_first = 1; tp.n = c->N;
        CU(c, qld_launch_fixed_table_fill(tp, c->rfix, c->N, c->s_copy));
        CU(c, qld_launch_digit_pack(c->rfix, c->N, c->N, c->K, c->digits, c->s_copy));
        c->launches += 2;
    } else if (!c->ring) {
        int rc = fill_tables(c, 1, c->N, c->s_copy);
        if (rc) return rc;
        if (c->tc_bins) {
            CU(c, qld_launch_bins_pack(static_cast<const int32_t *>(c->wtab), c->cap_w, c->rows_pad, c->N, c->digits, c->s_copy));
            c->launches++;
        }
    }
    CU(c, cudaEventRecord(c->tables_ev, c->s_copy));
    CU(c, cudaStreamWaitEvent(c->s_comp, c->tables_ev, 0));
    return QLD_OK;
}

// INT_BINS: the <= 16 combine weights sin / cos(2 pi r/den + phase) of the bin rows, computed on the device and kept in
// the by-value epilogue parameters
int fetch_bin_weights(qld_ctx *c)
{
    if (!c->is_int) return QLD_OK;
    TableFillParams tp;
    memset(&tp, 0, sizeof tp);
    tp.K = c->K; tp.is_int = 1; tp.rows = c->rows_pad;
    for (int k = 0; k < c->K; ++k) tp.ref[k] = c->ref[k];
    double *scratch = reinterpret_cast<double *>(reinterpret_cast<unsigned char *>(c->tile_counter) + 256);
    CU(c, qld_launch_bin_weights(tp, scratch, c->s_copy));
    c->launches++;
    double w[2 * QLD_MAX_ROWS];
    CU(c, cudaMemcpyAsync(w, scratch, sizeof w, cudaMemcpyDeviceToHost, c->s_copy));
    CU(c, cudaStreamSynchronize(c->s_copy));
    for (int r = 0; r < QLD_MAX_ROWS; ++r) { c->fin.sw[r] = w[r]; c->fin.cw[r] = w[QLD_MAX_ROWS + r]; }
    return QLD_OK;
}

// the tile counter of the next persistent-kernel launch (zero) and the one that launch has to zero
void next_counters(qld_ctx *c, unsigned int **cur, unsigned int **nxt)
{
    // three counters in rotation: a launch that starts early (programmatic dependent launch, k_slide_bulk) zeroes a counter that the
    // launch still running before it does not use
    *cur = c->tile_counter + (c->counter_flip % 3u);
    *nxt = c->tile_counter + ((c->counter_flip + 1u) % 3u);
    c->counter_flip++;
}

// make the copy stream wait for demods that still read frames <= last_overwritten
int wait_for_readers(qld_ctx *c, int64_t last_overwritten)
{
    int best = -1;
    for (int i = 0; i < N_DEMOD_EVENTS; ++i) {
        const int idx = (c->demod_ev_next + i) % N_DEMOD_EVENTS;   // oldest .. newest: keep the newest reader
        if (c->demod_ev[idx].used && c->demod_ev[idx].oldest_read <= last_overwritten) best = idx;
    }
    if (best >= 0) CU(c, cudaStreamWaitEvent(c->s_copy, c->demod_ev[best].ev, 0));
    return QLD_OK;
}

// src == NULL: the frames were written in place by the caller (qld_commit_frames); nothing is copied
int push_common(qld_ctx *c, const void *src, int n, cudaMemcpyKind kind, bool producer_wait = false)
{
    const size_t fb = (size_t)c->HW * c->bytes;
    bool enqueued = src != nullptr || producer_wait || !c->ring;
    if (!c->ring) {
        if (c->pushed + n > c->N) return fail(c, QLD_E_OVERRUN, "push: whole-window store already holds N frames (qld_reset first)");
        // frames still being read by an earlier demod of the previous stack
        int rc = wait_for_readers(c, INT64_MAX);
        if (rc) return rc;
        if (src) CU(c, cudaMemcpyAsync(c->frames + (size_t)c->pushed * fb, src, (size_t)n * fb, kind, c->s_copy));
    } else {
        const int64_t first = c->pushed + 1, last = c->pushed + n;
        const int64_t oldest_needed = c->seeded ? c->win_start + 1 : 1;
        if (last - c->cap >= oldest_needed) return fail(c, QLD_E_OVERRUN, "push: would overwrite frames a pending window still needs");
        if (last - c->cap >= 1) {
            int rc = wait_for_readers(c, last - c->cap);
            if (rc) return rc;
        }
        const int slot = (int)((first - 1) % c->cap);
        const int n1 = n < c->cap - slot ? n : c->cap - slot;
        if (src) {
            CU(c, cudaMemcpyAsync(c->frames + (size_t)slot * fb, src, (size_t)n1 * fb, kind, c->s_copy));
            if (n1 < n) CU(c, cudaMemcpyAsync(c->frames, static_cast<const unsigned char *>(src) + (size_t)n1 * fb, (size_t)(n - n1) * fb, kind, c->s_copy));
        }
        if (last > c->tab_filled) {
            // The table entry of a frame depends on its index only, so the tables may run ahead of the frames as far as the
            // table ring allows: an entry may be overwritten once no issued or pending window needs it (a window that starts
            // after a frames reads the entries of frames a .. a + N).  With a roomy ring most pushes then launch nothing.
            int64_t floor_needed = c->seeded ? c->win_start : 0;
            for (int i = 0; i < N_DEMOD_EVENTS; ++i)
                if (c->demod_ev[i].used && c->demod_ev[i].oldest_read - 1 < floor_needed) floor_needed = c->demod_ev[i].oldest_read - 1;
            int64_t target = floor_needed + c->cap_w - 1;
            if (target > last + 4096) target = last + 4096;
            if (target < last) target = last;                 // the frames themselves always fit (checked above)
            int rc = fill_tables(c, c->tab_filled + 1, (int)(target - c->tab_filled), c->s_copy);
            if (rc) return rc;
            c->tab_filled = target;
            enqueued = true;
        }
    }
    c->pushed += n;
    if (enqueued) {                                           // nothing new on the copy stream: the last event still stands
        cudaEvent_t ev = c->push_ev[c->push_ev_next];
        c->push_ev_next = (c->push_ev_next + 1) % N_PUSH_EVENTS;
        CU(c, cudaEventRecord(ev, c->s_copy));
        c->push_seq++;
        c->push_pending = true;
    }
    return QLD_OK;
}

cudaEvent_t last_push_event(qld_ctx *c) { return c->push_ev[(c->push_ev_next + N_PUSH_EVENTS - 1) % N_PUSH_EVENTS]; }

FinParams fin_with_maps(const qld_ctx *c)
{
    FinParams f = c->fin;
    f.I = c->mapI; f.Q = c->mapQ; f.amp = c->mapA; f.phase = c->mapP;
    f.rot = (c->window_relative && c->ring) ? reinterpret_cast<const double *>(reinterpret_cast<const unsigned char *>(c->tile_counter) + 256) : nullptr;
    return f;
}

// window-relative maps: the rotation factors of the window that starts after `a` frames, ahead of the demod kernel
int set_window_rotation(qld_ctx *c, int64_t a)
{
    if (!(c->window_relative && c->ring)) return QLD_OK;
    TableFillParams tp;
    memset(&tp, 0, sizeof tp);
    tp.K = c->K;
    for (int k = 0; k < c->K; ++k) tp.ref[k] = c->ref[k];
    double *rot = reinterpret_cast<double *>(reinterpret_cast<unsigned char *>(c->tile_counter) + 256);
    CU(c, qld_launch_window_rotation(tp, a, rot, c->s_comp));
    c->launches++;
    return QLD_OK;
}

int record_demod(qld_ctx *c, int64_t oldest_read)
{
    DemodEvent &d = c->demod_ev[c->demod_ev_next];
    c->demod_ev_next = (c->demod_ev_next + 1) % N_DEMOD_EVENTS;
    // Only the last N_DEMOD_EVENTS launches are remembered, and the host is never throttled: on a roomy ring it can be more
    // launches than that ahead of the GPU.  A launch about to be forgotten may still be queued; what it reads (frames: wait_for_readers,
    // table entries: the look-ahead in push_common) is protected only while it is remembered.  So the copy stream is held behind it
    // before its slot is reused: nothing the copy stream is given from here on can overtake a launch older than the remembered ones.
    if (d.used) CU(c, cudaStreamWaitEvent(c->s_copy, d.ev, 0));
    d.oldest_read = oldest_read; d.used = true;
    CU(c, cudaEventRecord(d.ev, c->s_comp));
    return QLD_OK;
}

// frames first+1 .. first+n (0-based offset `first`) as runs of consecutive store slots; returns the new run count
int add_runs(const qld_ctx *c, DemodRun *runs, int at, int64_t first, int n, int sign)
{
    const int slot = (int)(first % c->cap);
    const int n0 = n < c->cap - slot ? n : c->cap - slot;
    runs[at].slot0 = slot; runs[at].n = n0; runs[at].w0 = (int)((first + 1) % c->cap_w); runs[at].sign = sign;
    ++at;
    if (n0 < n) {
        runs[at].slot0 = 0; runs[at].n = n - n0; runs[at].w0 = (int)((first + 1 + n0) % c->cap_w); runs[at].sign = sign;
        ++at;
    }
    return at;
}

int stream_tmap_for(qld_ctx *c, const StreamShape &sh)
{
    if (c->stream_tmap_frames != c->frames || sh.seg != c->stream_shape.seg || sh.kc != c->stream_shape.kc) {
        CU(c, qld_stream_encode_tmap(c->stream_tmap, c->frames, c->HW * c->bytes, c->cap, sh));
        c->stream_tmap_frames = c->frames;
        c->stream_shape = sh;
    }
    return QLD_OK;
}

// The fields every launch over the ring / store shares: the store, the tables, the stored sums, the epilogue.  a_win = frames
// before the window the launch finalises (for the pedestal sums of the fp32 mode).
DemodParams base_params(const qld_ctx *c, int64_t a_win)
{
    DemodParams p;
    memset(&p, 0, sizeof p);
    p.big_endian = c->big_endian;
    p.frames = c->frames; p.frame_stride = c->HW * c->bytes; p.HW = c->HW;
    p.cap = c->cap; p.cap_w = c->cap_w;
    p.cum_lo = (int)(a_win % c->cap_w); p.cum_hi = (int)((a_win + c->N) % c->cap_w);
    p.wtab = c->wtab; p.cum = c->cum;
    p.onehot = c->is_int && c->K == 1 && c->ref[0].use_diff != 2;
    p.fin = fin_with_maps(c);
    return p;
}

// one k_demod_stream launch with the next pair of tile counters
int launch_stream(qld_ctx *c, const DemodParams &p, const StreamShape &sh)
{
    int rc = stream_tmap_for(c, sh);
    if (rc) return rc;
    unsigned int *cur, *nxt;
    next_counters(c, &cur, &nxt);
    CU(c, qld_launch_demod_stream(c->dtype, c->is_int, c->rows_pad, c->stream_tmap, p, sh, cur, nxt, c->n_sms, c->s_comp));
    c->launches++;
    c->last_kernel = "k_demod_stream";
    return QLD_OK;
}

// whole-window kernel over absolute frames a+1 .. a+N; seeds the sliding accumulators when asked
int run_whole_tc(qld_ctx *c)
{
    if (!c->tmap_valid) {
        CU(c, qld_tc_encode_tmap(c->tmap, c->frames, c->HW * c->bytes, c->N, c->K, c->n_sms, c->dbg_tc));
        c->tmap_valid = true;
    }
    TcParams p;
    memset(&p, 0, sizeof p);
    p.HW = c->HW; p.row_bytes = c->HW * c->bytes; p.N = c->N; p.bytes = c->bytes; p.big_endian = c->big_endian;
    p.digits = c->digits; p.sums_out = c->sums;
    next_counters(c, &p.tile_counter, &p.tile_counter_next);
    p.force_T = c->dbg_tc[0]; p.force_stages = c->dbg_tc[1]; p.force_kc = c->dbg_tc[2];
    p.fin = fin_with_maps(c);
    CU(c, qld_launch_demod_tc(c->tmap, p, c->n_sms, c->s_comp));
    c->launches++;
    c->last_kernel = "k_demod_tc";
    return record_demod(c, 1);
}

// INT_BINS whole window as a one-digit int8 contraction (A3' on the tensor cores): exact int32 bins into the accumulator rows
int run_whole_tc_bins(qld_ctx *c)
{
    if (!c->tmap_valid) {
        CU(c, qld_tc_encode_tmap(c->tmap, c->frames, c->HW * c->bytes, c->N, 2 /* 16 columns */, c->n_sms, c->dbg_tc));
        c->tmap_valid = true;
    }
    TcParams p;
    memset(&p, 0, sizeof p);
    p.HW = c->HW; p.row_bytes = c->HW * c->bytes; p.N = c->N; p.bytes = c->bytes; p.big_endian = c->big_endian;
    p.digits = c->digits;
    next_counters(c, &p.tile_counter, &p.tile_counter_next);
    p.force_T = c->dbg_tc[0]; p.force_stages = c->dbg_tc[1]; p.force_kc = c->dbg_tc[2];
    p.bins_rows = c->rows_pad; p.bins_out = static_cast<int32_t *>(c->acc); p.bins_stride = c->HW;
    p.fin = fin_with_maps(c);
    CU(c, qld_launch_demod_tc(c->tmap, p, c->n_sms, c->s_comp));
    c->launches++;
    c->last_kernel = "k_demod_tc";
    return record_demod(c, 1);
}

int run_whole(qld_ctx *c, int64_t a, bool seed)
{
    if (c->is_fixed) return run_whole_tc(c);
    if (c->tc_bins && !seed && (reinterpret_cast<uintptr_t>(c->frames) & 15) == 0) {
        // frames large enough for the streaming kernels (or a forced tensor-core tile shape): the contraction is 2.5x faster
        // than the CUDA-core bins on an L2-resident stack and as fast as HBM on a large one
        const StreamShape big = qld_stream_shape(c->dtype, 1, c->rows_pad, c->HW, c->frames, c->n_sms, 0, 0);
        if (c->dbg_tc[0] > 0 || (big.seg > 0 && c->dbg_stream[0] == 0)) return run_whole_tc_bins(c);
    }
    DemodParams p = base_params(c, a);
    p.slot0 = (int)(a % c->cap); p.n = c->N;
    p.w0 = (int)((a + 1) % c->cap_w);
    p.acc_out = (seed || c->is_int) ? c->acc : nullptr;
    p.ped_out = (seed && !c->is_int) ? c->ped : nullptr;
    p.n_runs = add_runs(c, p.run, 0, a, c->N, +1);
    // large, 16-byte-aligned frames: the TMA-fed persistent kernel; otherwise the register-staged one
    const StreamShape sh = qld_stream_shape(c->dtype, c->is_int, c->rows_pad, c->HW, c->frames, c->n_sms, c->dbg_stream[0], c->dbg_stream[1]);
    if (sh.seg > 0) {
        const int rc = launch_stream(c, p, sh);
        return rc ? rc : record_demod(c, a + 1);
    }
    CU(c, qld_launch_demod_whole(c->dtype, c->is_int, c->rows_pad, p, c->s_comp));
    c->last_kernel = "k_demod_whole";
    c->launches++;
    return record_demod(c, a + 1);
}

// The sliding update through k_slide_bulk when the frames are large enough (or forced): returns 1 if it was launched,
// 0 if the kernel does not apply, < 0 on error.
int try_slide_bulk(qld_ctx *c, const DemodParams &p)
{
    const int n_map_rows = c->K * ((c->mapI != nullptr) + (c->mapQ != nullptr) + (c->mapA != nullptr) + (c->mapP != nullptr));
    const int kind = c->is_int ? 1 : (c->fix_ring ? 2 : 0);
    const SlideShape sh = qld_slide_shape(c->dtype, kind, c->rows_pad, p.part != nullptr, n_map_rows, c->HW, c->frames, c->n_sms, c->fix_ring ? 1 : c->dbg_slide);
    if (sh.seg == 0) return 0;
    if (c->slide_tmap_frames != c->frames || sh.seg != c->slide_shape.seg || sh.kc != c->slide_shape.kc) {
        cudaError_t e = qld_slide_encode_tmap(c->slide_tmap, c->frames, c->HW * c->bytes, c->cap, sh);
        if (e != cudaSuccess) return cuda_fail(c, e, "qld_slide_encode_tmap");
        c->slide_tmap_frames = c->frames;
        c->slide_shape = sh;
    }
    unsigned int *cur, *nxt;
    next_counters(c, &cur, &nxt);
    cudaError_t e = qld_launch_slide_bulk(c->dtype, kind, c->rows_pad, c->slide_tmap, p, sh, cur, nxt, c->n_sms, c->s_comp);
    if (e != cudaSuccess) return cuda_fail(c, e, "qld_launch_slide_bulk");
    c->launches++;
    c->last_kernel = "k_slide_bulk";
    return 1;
}

// Block-partial mode (8(f3)): one launch over the frames of batch b of the window that starts at offset a.
// sub = false: seeding (the slot is only written); sub = true: a sliding update (the slot's old content is the
// expired batch: taken off the accumulators, then overwritten).
int run_partial_batch(qld_ctx *c, int64_t a_win, int64_t first, int slot, bool add, bool sub, bool first_of_seed)
{
    DemodParams p = base_params(c, a_win);
    p.acc_out = c->acc; p.acc_add = add ? 1 : 0;
    p.part = c->part + (size_t)slot * c->rows_pad * c->HW * (c->is_int ? 4 : 8);
    p.part_sub = sub ? 1 : 0;
    p.n_runs = add_runs(c, p.run, 0, first, c->slide_hop, +1);
    if (add && sub) {                                       // steady state: every byte through the copy engines
        DemodParams q = p;
        q.ped_in = c->is_int ? nullptr : c->ped;
        const int rc = try_slide_bulk(c, q);
        if (rc != 0) return rc < 0 ? rc : QLD_OK;
    }
    if (c->fix_ring) return fail(c, QLD_E_UNSUPPORTED, "FIXED on a ring: the state of a tile does not fit the bulk-copy kernel's shared memory");
    const StreamShape sh = qld_stream_shape(c->dtype, c->is_int, c->rows_pad, c->HW, c->frames, c->n_sms, c->dbg_stream[0], c->dbg_stream[1]);
    if (sh.seg == 0 || c->slide_hop < sh.kc) return fail(c, QLD_E_UNSUPPORTED, "slide_hop: frames too small / hop too short for the TMA kernel");
    if (!c->is_int) {
        if (first_of_seed) p.ped_out = c->ped; else p.ped_in = c->ped;
    }
    return launch_stream(c, p, sh);
}

// window a+1 .. a+N from scratch: the sums, and (block-partial mode) the N/hop per-batch partials
// FIXED on a ring: the window from scratch through k_slide_bulk -- the stored sums (and partial sums) are zeroed and the
// window's frames are "added" to them
int seed_fix_ring(qld_ctx *c, int64_t a)
{
    const size_t rowset = (size_t)c->rows_pad * c->HW * 8;
    CU(c, cudaMemsetAsync(c->acc, 0, rowset, c->s_comp));
    if (c->slide_hop > 0) CU(c, cudaMemsetAsync(c->part, 0, rowset * c->n_part, c->s_comp));
    const int n_launch = c->slide_hop > 0 ? c->n_part : 1;
    for (int b = 0; b < n_launch; ++b) {
        DemodParams q = base_params(c, a);
        q.acc_out = c->acc; q.acc_add = 1;
        if (c->slide_hop > 0) {
            q.part = c->part + (size_t)b * rowset;
            q.part_sub = 1;
            q.n_runs = add_runs(c, q.run, 0, a + (int64_t)b * c->slide_hop, c->slide_hop, +1);
        } else {
            q.n_runs = add_runs(c, q.run, 0, a, c->N, +1);
        }
        const int rc = try_slide_bulk(c, q);
        if (rc < 0) return rc;
        if (rc == 0) return fail(c, QLD_E_UNSUPPORTED, "FIXED on a ring: the state of a tile does not fit the bulk-copy kernel's shared memory");
    }
    return record_demod(c, a + 1);
}

int seed_window(qld_ctx *c, int64_t a)
{
    if (c->fix_ring) return seed_fix_ring(c, a);
    if (c->slide_hop == 0) return run_whole(c, a, true);
    for (int b = 0; b < c->n_part; ++b) {
        int rc = run_partial_batch(c, a, a + (int64_t)b * c->slide_hop, b, b > 0, false, b == 0);
        if (rc) return rc;
    }
    return record_demod(c, a + 1);
}

int run_slide(qld_ctx *c, int64_t a_old, int hop)
{
    const int64_t a_new = a_old + hop;
    if (c->slide_hop > 0) {
        // the expired batch and the new one share a slot: batch j of the seeded window lives in slot j mod M
        const int slot = (int)(c->hops_since_seed % c->n_part);
        int rc = run_partial_batch(c, a_new, a_old + c->N, slot, true, true, false);
        if (rc) return rc;
        return record_demod(c, a_old + 1);                    // conservative: the whole window stays protected from overwriting
    }
    // {expired, -w} + {new, +w} added to the stored sums
    DemodParams q = base_params(c, a_new);
    q.acc_out = c->acc; q.acc_add = 1;
    q.ped_in = c->is_int ? nullptr : c->ped;
    {
        const int n = add_runs(c, q.run, 0, a_old, hop, -1);        // expired: frames a_old+1 .. a_old+hop
        q.n_runs = add_runs(c, q.run, n, a_old + c->N, hop, +1);   // new: frames a_old+N+1 .. a_old+N+hop
    }
    {
        const int rc = try_slide_bulk(c, q);                       // k_slide_bulk when the frames are large enough
        if (rc != 0) return rc < 0 ? rc : record_demod(c, a_old + 1);
        if (c->fix_ring) return fail(c, QLD_E_UNSUPPORTED, "FIXED on a ring: the state of a tile does not fit the bulk-copy kernel's shared memory");
    }
    // smaller frames, hops of at least one pipeline stage: the TMA-fed whole-window kernel over the same run list
    const StreamShape sh = qld_stream_shape(c->dtype, c->is_int, c->rows_pad, c->HW, c->frames, c->n_sms, c->dbg_stream[0], c->dbg_stream[1]);
    if (sh.seg > 0 && hop >= sh.kc) {
        const int rc = launch_stream(c, q, sh);
        return rc ? rc : record_demod(c, a_old + 1);
    }
    SlideParams p;
    memset(&p, 0, sizeof p);
    p.big_endian = c->big_endian;
    p.frames = c->frames; p.frame_stride = c->HW * c->bytes; p.HW = c->HW;
    p.cap = c->cap; p.cap_w = c->cap_w; p.hop = hop;
    p.new_slot0 = (int)((a_old + c->N) % c->cap);          // first new frame is a_old+N+1 -> slot (a_old+N) mod cap
    p.old_slot0 = (int)(a_old % c->cap);                   // first expired frame is a_old+1
    p.new_w0 = (int)((a_old + c->N + 1) % c->cap_w);
    p.old_w0 = (int)((a_old + 1) % c->cap_w);
    p.cum_lo = (int)(a_new % c->cap_w); p.cum_hi = (int)((a_new + c->N) % c->cap_w);
    p.wtab = c->wtab; p.cum = c->cum; p.acc = c->acc; p.ped = c->ped;
    p.fin = fin_with_maps(c);
    CU(c, qld_launch_demod_slide(c->dtype, c->is_int, c->rows_pad, p, c->s_comp));
    c->launches++;
    c->last_kernel = "k_demod_slide";
    return record_demod(c, a_old + 1);
}

}  // namespace

extern "C" {

int qld_workspace_bytes(const qld_config *cfg, size_t *bytes_out)
{
    Plan pl;
    std::string err;
    int rc = make_plan(cfg, &pl, &err);
    if (rc) { g_create_error = err; return rc; }
    if (!bytes_out) return fail(nullptr, QLD_E_INVAL, "bytes_out is NULL");
    *bytes_out = pl.total;
    return QLD_OK;
}

int qld_create(const qld_config *cfg, qld_ctx **ctx_out)
{
    if (!ctx_out) return fail(nullptr, QLD_E_INVAL, "ctx_out is NULL");
    *ctx_out = nullptr;
    Plan pl;
    std::string err;
    int rc = make_plan(cfg, &pl, &err);
    if (rc) { g_create_error = err; return rc; }
    int ndev = 0;
    cudaError_t ce = cudaGetDeviceCount(&ndev);
    if (ce != cudaSuccess || ndev < 1) {
        (void)cudaGetLastError();
        return fail(nullptr, QLD_E_CUDA, "no CUDA device: this library has no CPU fallback");
    }
    qld_ctx *c = new (std::nothrow) qld_ctx();
    if (!c) return fail(nullptr, QLD_E_NOMEM, "host allocation failed");
    c->H = pl.H; c->W = pl.W; c->dtype = pl.dtype; c->bytes = pl.bytes; c->N = pl.N; c->K = pl.K;
    c->big_endian = pl.dtype == QLD_U16_BE ? 1 : 0;
    c->window_relative = cfg->window_relative == 1;
    c->accum = pl.accum; c->norm = pl.norm; c->maps = pl.maps; c->resync_hops = cfg->resync_hops;
    c->HW = pl.HW; c->max_value = cfg->max_value; c->cap = pl.cap; c->cap_w = pl.cap_w;
    c->ring = pl.ring; c->external = pl.external; c->is_int = pl.is_int; c->is_fixed = pl.is_fixed; c->fix_ring = pl.fix_ring; c->tc_bins = pl.tc_bins; c->rows = pl.rows; c->rows_pad = pl.rows_pad;
    for (int k = 0; k < pl.K; ++k) c->ref[k] = pl.ref[k];
    c->fin = pl.fin;
    c->ws_bytes = pl.total;
    c->tables_supplied = cfg->ref_tables_supplied == 1;
    auto cleanup = [&](int code) { qld_destroy(c); return code; };
    if (cfg->workspace) {
        if (cfg->workspace_bytes < pl.total || (reinterpret_cast<uintptr_t>(cfg->workspace) & 255)) {
            delete c;
            return fail(nullptr, QLD_E_NOMEM, "caller workspace too small or not 256-byte aligned");
        }
        c->ws = cfg->workspace; c->own_ws = false;
    } else {
        ce = cudaMalloc(&c->ws, pl.total);
        if (ce != cudaSuccess) { (void)cudaGetLastError(); delete c; return fail(nullptr, QLD_E_NOMEM, "cudaMalloc of the workspace failed"); }
        c->own_ws = true;
    }
    unsigned char *b = static_cast<unsigned char *>(c->ws);
    c->frames = pl.external ? nullptr : b + pl.off_frames;
    c->own_frames = c->frames;
    c->wtab = b + pl.off_wtab; c->cum = reinterpret_cast<double *>(b + pl.off_cum);
    c->acc = b + pl.off_acc; c->ped = reinterpret_cast<float *>(b + pl.off_ped);
    c->part = b + pl.off_part; c->slide_hop = pl.slide_hop; c->n_part = pl.slide_hop > 0 ? pl.N / pl.slide_hop : 0;
    c->mapI = (pl.maps & QLD_MAP_I) ? reinterpret_cast<float *>(b + pl.off_I) : nullptr;
    c->mapQ = (pl.maps & QLD_MAP_Q) ? reinterpret_cast<float *>(b + pl.off_Q) : nullptr;
    c->mapA = (pl.maps & QLD_MAP_AMP) ? reinterpret_cast<float *>(b + pl.off_A) : nullptr;
    c->mapP = (pl.maps & QLD_MAP_PHASE) ? reinterpret_cast<float *>(b + pl.off_P) : nullptr;
    c->tile_counter = reinterpret_cast<unsigned int *>(b + pl.off_counter);
    {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&c->n_sms, cudaDevAttrMultiProcessorCount, dev);
    }
    if (pl.tc_bins) c->digits = reinterpret_cast<int8_t *>(b + pl.off_digits);
    if (pl.is_fixed) {
        c->rfix = reinterpret_cast<int32_t *>(b + pl.off_rfix);
        c->digits = reinterpret_cast<int8_t *>(b + pl.off_digits);
        c->sums = (pl.maps & QLD_MAP_SUMS_I64) ? reinterpret_cast<int64_t *>(b + pl.off_sums) : nullptr;
        if ((reinterpret_cast<uintptr_t>(c->frames) & 15) != 0) { if (c->own_ws) cudaFree(c->ws); delete c; return fail(nullptr, QLD_E_NOMEM, "workspace not 16-byte aligned"); }
    }

    c->s_comp = static_cast<cudaStream_t>(cfg->compute_stream);
    c->s_copy = static_cast<cudaStream_t>(cfg->copy_stream);
    if (!c->s_comp) { if (cudaStreamCreateWithFlags(&c->s_comp, cudaStreamNonBlocking) != cudaSuccess) return cleanup(fail(nullptr, QLD_E_CUDA, "stream creation failed")); c->own_comp = true; }
    if (!c->s_copy) { if (cudaStreamCreateWithFlags(&c->s_copy, cudaStreamNonBlocking) != cudaSuccess) return cleanup(fail(nullptr, QLD_E_CUDA, "stream creation failed")); c->own_copy = true; }
    for (int i = 0; i < N_PUSH_EVENTS; ++i)
        if (cudaEventCreateWithFlags(&c->push_ev[i], cudaEventDisableTiming) != cudaSuccess) return cleanup(fail(nullptr, QLD_E_CUDA, "event creation failed"));
    for (int i = 0; i < N_DEMOD_EVENTS; ++i) {
        if (cudaEventCreateWithFlags(&c->demod_ev[i].ev, cudaEventDisableTiming) != cudaSuccess) return cleanup(fail(nullptr, QLD_E_CUDA, "event creation failed"));
        c->demod_ev[i].used = false;
    }
    if (cudaEventCreateWithFlags(&c->tables_ev, cudaEventDisableTiming) != cudaSuccess) return cleanup(fail(nullptr, QLD_E_CUDA, "event creation failed"));
    rc = init_device_state(c);
    if (rc == QLD_OK) rc = fetch_bin_weights(c);
    if (rc) { g_create_error = c->err; return cleanup(rc); }
    ce = cudaStreamSynchronize(c->s_copy);
    if (ce != cudaSuccess) { g_create_error = cudaGetErrorString(ce); return cleanup(QLD_E_CUDA); }
    *ctx_out = c;
    return QLD_OK;
}

static int push_checked(qld_ctx *c, const void *src, int n, cudaMemcpyKind kind)
{
    NvtxRange nvtx("qld_push_frames");
    if (!c) return QLD_E_INVAL;
    if (c->sticky) return QLD_E_CUDA;
    if (!src || n < 1) return fail(c, QLD_E_INVAL, "push: null buffer or n_frames < 1");
    if (c->external) return fail(c, QLD_E_STATE, "push: this context takes frames in place (external_store): attach + qld_commit_frames");
    if (c->frames != c->own_frames) return fail(c, QLD_E_STATE, "push: a caller buffer is attached in place of the store (qld_reset detaches it)");
    if (n > c->cap) return fail(c, QLD_E_INVAL, "push: more frames than the store holds");
    return push_common(c, src, n, kind);
}

int qld_push_frames(qld_ctx *c, const void *host_frames, int n_frames) { return push_checked(c, host_frames, n_frames, cudaMemcpyHostToDevice); }

int qld_push_frames_device(qld_ctx *c, const void *device_frames, int n_frames) { return push_checked(c, device_frames, n_frames, cudaMemcpyDeviceToDevice); }

int qld_commit_frames(qld_ctx *c, int n_frames, void *producer_stream)
{
    NvtxRange nvtx("qld_commit_frames");
    if (!c) return QLD_E_INVAL;
    if (c->sticky) return QLD_E_CUDA;
    if (!c->external) return fail(c, QLD_E_STATE, "commit: context owns its frame store (use qld_push_frames)");
    if (!c->frames) return fail(c, QLD_E_STATE, "commit: no frame store attached");
    if (n_frames < 1 || n_frames > c->cap) return fail(c, QLD_E_INVAL, "commit: n_frames must be 1..capacity");
    if (producer_stream) {
        // tables and later demods are ordered after the producer's writes
        CU(c, cudaEventRecord(c->tables_ev, static_cast<cudaStream_t>(producer_stream)));
        CU(c, cudaStreamWaitEvent(c->s_copy, c->tables_ev, 0));
    }
    return push_common(c, nullptr, n_frames, cudaMemcpyDefault, producer_stream != nullptr);
}

int qld_attach_frames_device(qld_ctx *c, const void *device_frames)
{
    if (!c) return QLD_E_INVAL;
    if (c->sticky) return QLD_E_CUDA;
    if (!device_frames) return fail(c, QLD_E_INVAL, "attach: null buffer");
    if (c->ring && !c->external) return fail(c, QLD_E_STATE, "attach: this ring context owns its frame store (create it with external_store = 1)");
    if (c->pushed > 0 && c->ring) return fail(c, QLD_E_STATE, "attach: ring already holds frames (qld_reset first)");
    if (c->is_fixed && (reinterpret_cast<uintptr_t>(device_frames) & 15)) return fail(c, QLD_E_INVAL, "attach: FIXED accumulation needs a 16-byte aligned buffer");
    c->frames = const_cast<unsigned char *>(static_cast<const unsigned char *>(device_frames));
    c->tmap_valid = false;
    if (!c->ring) c->pushed = c->N;
    return QLD_OK;
}

int qld_push_done(qld_ctx *c, int block)
{
    if (!c) return QLD_E_INVAL;
    if (!c->push_pending) return QLD_OK;
    cudaEvent_t ev = last_push_event(c);
    if (block) { CU(c, cudaEventSynchronize(ev)); c->push_pending = false; return QLD_OK; }
    cudaError_t e = cudaEventQuery(ev);
    if (e == cudaSuccess) { c->push_pending = false; return QLD_OK; }
    if (e == cudaErrorNotReady) return QLD_E_STATE;
    return cuda_fail(c, e, "cudaEventQuery");
}

int qld_demod(qld_ctx *c, int mode, int hop)
{
    NvtxRange nvtx(mode == QLD_SLIDE ? "qld_demod(SLIDE)" : "qld_demod(WHOLE)");
    if (!c) return QLD_E_INVAL;
    if (c->sticky) return QLD_E_CUDA;
    if (mode != QLD_WHOLE && mode != QLD_SLIDE) return fail(c, QLD_E_INVAL, "demod: unknown mode");
    if (!c->frames) return fail(c, QLD_E_STATE, "demod: no frames attached");
    if (c->tables_supplied && c->tables_set != (1u << c->K) - 1u) return fail(c, QLD_E_STATE, "demod: qld_set_ref_tables has not been called for every reference");
    if (c->push_seq != c->waited_seq) {                      // order the kernels after every push issued so far (once per event)
        CU(c, cudaStreamWaitEvent(c->s_comp, last_push_event(c), 0));
        c->waited_seq = c->push_seq;
    }
    if (mode == QLD_WHOLE) {
        if (c->pushed < c->N) return fail(c, QLD_E_STATE, "demod: fewer than N frames stored");
        const int64_t a = c->ring ? c->pushed - c->N : 0;
        int rc = set_window_rotation(c, a);
        if (rc == QLD_OK) rc = c->ring ? seed_window(c, a) : run_whole(c, a, false);
        if (rc) return rc;
        if (c->ring) { c->seeded = true; c->win_start = a; c->hops_since_seed = 0; }
        c->windows_done++;
        return QLD_OK;
    }
    if (!c->ring) return fail(c, QLD_E_STATE, "demod: QLD_SLIDE needs a ring context (ring_frames > N)");
    if (!c->seeded) {
        if (c->pushed < c->N) return fail(c, QLD_E_STATE, "demod: fewer than N frames pushed");
        int rc = set_window_rotation(c, 0);
        if (rc == QLD_OK) rc = seed_window(c, 0);
        if (rc) return rc;
        c->seeded = true; c->win_start = 0; c->hops_since_seed = 0; c->windows_done++;
        return QLD_OK;
    }
    if (hop < 1 || hop > c->N) return fail(c, QLD_E_INVAL, "demod: hop must be 1..N");
    if (c->slide_hop > 0 && hop != c->slide_hop) return fail(c, QLD_E_INVAL, "demod: this context slides by cfg.slide_hop only");
    if (c->pushed < c->win_start + hop + c->N) return fail(c, QLD_E_STATE, "demod: fewer than hop new frames pushed");
    int rc = set_window_rotation(c, c->win_start + hop);
    if (rc) return rc;
    // FP32 ring sums random-walk away from a recompute (each hop adds rounding of its own): resynchronise from the ring
    // every resync_hops hops; 0 = automatic (16 windows' worth of hops: 1/16 more traffic), negative = never
    const int64_t resync = c->resync_hops > 0 ? c->resync_hops : (c->resync_hops == 0 ? 16 * (int64_t)((c->N + hop - 1) / hop) : 0);
    if (!c->is_int && !c->fix_ring && resync > 0 && c->hops_since_seed + 1 >= resync) {
        rc = seed_window(c, c->win_start + hop);
        c->hops_since_seed = 0;
    } else {
        rc = run_slide(c, c->win_start, hop);
        c->hops_since_seed++;
    }
    if (rc) return rc;
    c->win_start += hop;
    c->windows_done++;
    return QLD_OK;
}

int qld_get_maps(qld_ctx *c, int k, const float **I, const float **Q, const float **amp, const float **phase)
{
    if (!c || k < 0 || k >= c->K) return c ? fail(c, QLD_E_INVAL, "get_maps: k out of range") : QLD_E_INVAL;
    const size_t o = (size_t)k * c->HW;
    if (I) *I = c->mapI ? c->mapI + o : nullptr;
    if (Q) *Q = c->mapQ ? c->mapQ + o : nullptr;
    if (amp) *amp = c->mapA ? c->mapA + o : nullptr;
    if (phase) *phase = c->mapP ? c->mapP + o : nullptr;
    return QLD_OK;
}

int qld_get_bins(qld_ctx *c, int k, const int32_t **rows, int *n_rows)
{
    if (!c || k < 0 || k >= c->K) return c ? fail(c, QLD_E_INVAL, "get_bins: k out of range") : QLD_E_INVAL;
    if (!c->is_int) return fail(c, QLD_E_STATE, "get_bins: context does not accumulate integer bins");
    if (rows) *rows = static_cast<const int32_t *>(c->acc) + (size_t)c->ref[k].row_off * c->HW;
    if (n_rows) *n_rows = c->ref[k].n_rows;
    return QLD_OK;
}

int qld_read_map(qld_ctx *c, int k, int which, float *host_dst)
{
    NvtxRange nvtx("qld_read_map");
    if (!c || !host_dst || k < 0 || k >= c->K) return c ? fail(c, QLD_E_INVAL, "read_map: bad argument") : QLD_E_INVAL;
    if (c->sticky) return QLD_E_CUDA;
    const float *src = which == QLD_MAP_I ? c->mapI : which == QLD_MAP_Q ? c->mapQ : which == QLD_MAP_AMP ? c->mapA : which == QLD_MAP_PHASE ? c->mapP : nullptr;
    if (!src) return fail(c, QLD_E_INVAL, "read_map: map not produced by this context");
    CU(c, cudaMemcpyAsync(host_dst, src + (size_t)k * c->HW, (size_t)c->HW * 4, cudaMemcpyDeviceToHost, c->s_comp));
    return QLD_OK;
}

int qld_read_ref_table(qld_ctx *c, int k, int64_t s_first, int n, float *sin_out, float *cos_out)
{
    if (!c || k < 0 || k >= c->K || n < 1 || s_first < 1) return c ? fail(c, QLD_E_INVAL, "read_ref_table: bad argument") : QLD_E_INVAL;
    if (c->is_int || c->is_fixed || c->fix_ring) return fail(c, QLD_E_STATE, "read_ref_table: this context has no float table");
    if (c->ring && (s_first + n - 1 > c->pushed || s_first + c->cap_w <= (c->tab_filled > c->pushed ? c->tab_filled : c->pushed) + 1)) return fail(c, QLD_E_STATE, "read_ref_table: frames not in the ring");
    if (!c->ring && s_first + n - 1 > c->N) return fail(c, QLD_E_INVAL, "read_ref_table: beyond the window");
    CU(c, cudaStreamSynchronize(c->s_copy));
    for (int i = 0; i < n; ++i) {
        const int64_t e = (s_first + i) % c->cap_w;
        float w[2];
        CU(c, cudaMemcpy(w, static_cast<const float *>(c->wtab) + e * c->rows_pad + 2 * k, sizeof w, cudaMemcpyDeviceToHost));
        if (sin_out) sin_out[i] = w[0];
        if (cos_out) cos_out[i] = w[1];
    }
    return QLD_OK;
}

int qld_set_ref_tables(qld_ctx *c, int k, const double *sin_tab, const double *cos_tab, int64_t len)
{
    if (!c || k < 0 || k >= c->K || !sin_tab || !cos_tab) return c ? fail(c, QLD_E_INVAL, "set_ref_tables: bad argument") : QLD_E_INVAL;
    if (c->sticky) return QLD_E_CUDA;
    if (c->ring || c->is_int) return fail(c, QLD_E_UNSUPPORTED, "set_ref_tables: whole-window FP32 / FIXED contexts only");
    if (len != c->N) return fail(c, QLD_E_INVAL, "set_ref_tables: len must equal N");
    for (int64_t i = 0; i < len; ++i)
        if (!(sin_tab[i] >= -1.0 && sin_tab[i] <= 1.0 && cos_tab[i] >= -1.0 && cos_tab[i] <= 1.0))
            return fail(c, QLD_E_INVAL, "set_ref_tables: entries must lie in [-1, 1]");
    int rc = qld_sync(c);
    if (rc) return rc;
    double *tab = nullptr;
    if (cudaMalloc(&tab, (size_t)2 * len * sizeof(double)) != cudaSuccess) { (void)cudaGetLastError(); return fail(c, QLD_E_NOMEM, "set_ref_tables: device scratch"); }
    cudaError_t e = cudaMemcpy(tab, sin_tab, (size_t)len * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(tab + len, cos_tab, (size_t)len * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        if (c->is_fixed) {
            e = qld_launch_fixed_from_doubles(tab, (int)len, k, c->rfix, c->N, c->s_comp);
            if (e == cudaSuccess) e = qld_launch_digit_pack(c->rfix, c->N, c->N, c->K, c->digits, c->s_comp);
        } else {
            e = qld_launch_table_from_doubles(tab, (int)len, 2 * k, c->rows_pad, c->cap_w, c->wtab, c->cum, c->s_comp);
        }
        c->launches += c->is_fixed ? 2 : 1;
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->s_comp);
    cudaFree(tab);
    if (e != cudaSuccess) return cuda_fail(c, e, "set_ref_tables");
    c->tables_set |= 1u << k;
    return QLD_OK;
}

int qld_set_ref_table_fixed(qld_ctx *c, int k, const int32_t *sin_q30, const int32_t *cos_q30, int n)
{
    if (!c || k < 0 || k >= c->K || !sin_q30 || !cos_q30) return c ? fail(c, QLD_E_INVAL, "set_ref_table_fixed: bad argument") : QLD_E_INVAL;
    if (c->sticky) return QLD_E_CUDA;
    if (!c->is_fixed && !c->fix_ring) return fail(c, QLD_E_STATE, "set_ref_table_fixed: context does not use QLD_ACC_FIXED");
    if (c->fix_ring ? (n < 1 || n > c->pushed || n >= c->cap_w) : n != c->N)
        return fail(c, QLD_E_INVAL, c->fix_ring ? "set_ref_table_fixed: n must be 1 .. frames pushed (and fit the table ring)" : "set_ref_table_fixed: n must equal N");
    for (int i = 0; i < n; ++i)
        if (sin_q30[i] > (1 << 30) || sin_q30[i] < -(1 << 30) || cos_q30[i] > (1 << 30) || cos_q30[i] < -(1 << 30))
            return fail(c, QLD_E_INVAL, "set_ref_table_fixed: entries must lie in [-2^30, 2^30]");
    int rc = qld_sync(c);
    if (rc) return rc;
    if (c->fix_ring) {
        // ring: the entries of the n most recently pushed frames (absolute indices pushed-n+1 .. pushed), in place in the table ring
        int32_t *w = static_cast<int32_t *>(c->wtab);
        for (int i = 0; i < n; ++i) {
            const int64_t e = (c->pushed - n + 1 + i) % c->cap_w;
            const int32_t pair[2] = {sin_q30[i], cos_q30[i]};
            CU(c, cudaMemcpy(w + e * c->rows_pad + 2 * k, pair, sizeof pair, cudaMemcpyHostToDevice));
        }
        return QLD_OK;
    }
    CU(c, cudaMemcpy(c->rfix + (size_t)(2 * k) * c->N, sin_q30, (size_t)n * 4, cudaMemcpyHostToDevice));
    CU(c, cudaMemcpy(c->rfix + (size_t)(2 * k + 1) * c->N, cos_q30, (size_t)n * 4, cudaMemcpyHostToDevice));
    CU(c, qld_launch_digit_pack(c->rfix, c->N, c->N, c->K, c->digits, c->s_comp));
    c->launches++;
    c->tables_set |= 1u << k;
    return QLD_OK;
}

int qld_read_ref_table_fixed(qld_ctx *c, int k, int32_t *sin_q30, int32_t *cos_q30)
{
    if (!c || k < 0 || k >= c->K) return c ? fail(c, QLD_E_INVAL, "read_ref_table_fixed: bad argument") : QLD_E_INVAL;
    if (c->fix_ring) {                                       // ring: the entries of the N most recently pushed frames
        if (c->pushed < c->N) return fail(c, QLD_E_STATE, "read_ref_table_fixed: fewer than N frames pushed");
        int rc = qld_sync(c);
        if (rc) return rc;
        for (int i = 0; i < c->N; ++i) {
            const int64_t e = (c->pushed - c->N + 1 + i) % c->cap_w;
            int32_t w[2];
            CU(c, cudaMemcpy(w, static_cast<const int32_t *>(c->wtab) + e * c->rows_pad + 2 * k, sizeof w, cudaMemcpyDeviceToHost));
            if (sin_q30) sin_q30[i] = w[0];
            if (cos_q30) cos_q30[i] = w[1];
        }
        return QLD_OK;
    }
    if (!c->is_fixed) return fail(c, QLD_E_STATE, "read_ref_table_fixed: context does not use QLD_ACC_FIXED");
    int rc = qld_sync(c);
    if (rc) return rc;
    if (sin_q30) CU(c, cudaMemcpy(sin_q30, c->rfix + (size_t)(2 * k) * c->N, (size_t)c->N * 4, cudaMemcpyDeviceToHost));
    if (cos_q30) CU(c, cudaMemcpy(cos_q30, c->rfix + (size_t)(2 * k + 1) * c->N, (size_t)c->N * 4, cudaMemcpyDeviceToHost));
    return QLD_OK;
}

int qld_get_sums_i64(qld_ctx *c, int k, const int64_t **I, const int64_t **Q)
{
    if (!c || k < 0 || k >= c->K) return c ? fail(c, QLD_E_INVAL, "get_sums_i64: k out of range") : QLD_E_INVAL;
    if (c->fix_ring) {                                       // the stored sums of the current window are the exact int64 sums
        int64_t *a = static_cast<int64_t *>(c->acc);
        if (I) *I = a + (size_t)(2 * k) * c->HW;
        if (Q) *Q = a + (size_t)(2 * k + 1) * c->HW;
        return QLD_OK;
    }
    if (!c->sums) return fail(c, QLD_E_STATE, "get_sums_i64: needs QLD_ACC_FIXED and QLD_MAP_SUMS_I64");
    if (I) *I = c->sums + (size_t)(2 * k) * c->HW;
    if (Q) *Q = c->sums + (size_t)(2 * k + 1) * c->HW;
    return QLD_OK;
}

int qld_counters(const qld_ctx *c, int64_t *frames_pushed, int64_t *windows_done)
{
    if (!c) return QLD_E_INVAL;
    if (frames_pushed) *frames_pushed = c->pushed;
    if (windows_done) *windows_done = c->windows_done;
    return QLD_OK;
}

int qld_sync(qld_ctx *c)
{
    if (!c) return QLD_E_INVAL;
    CU(c, cudaStreamSynchronize(c->s_copy));
    CU(c, cudaStreamSynchronize(c->s_comp));
    c->push_pending = false;
    return QLD_OK;
}

int qld_reset(qld_ctx *c)
{
    if (!c) return QLD_E_INVAL;
    if (c->sticky) return QLD_E_CUDA;
    int rc = qld_sync(c);
    if (rc) return rc;
    c->pushed = 0; c->windows_done = 0; c->seeded = false; c->win_start = 0; c->hops_since_seed = 0; c->tab_filled = 0;
    for (int i = 0; i < N_DEMOD_EVENTS; ++i) c->demod_ev[i].used = false;
    if (!c->ring && c->frames != c->own_frames) {          // an attached stack is detached (an attached ring stays attached)
        c->frames = c->own_frames; c->tmap_valid = false; c->stream_tmap_frames = nullptr; c->slide_tmap_frames = nullptr;
    }
    if (c->ring) {
        rc = init_device_state(c);
        if (rc) return rc;
    }
    return QLD_OK;
}

void qld_destroy(qld_ctx *c)
{
    if (!c) return;
    if (c->s_copy) cudaStreamSynchronize(c->s_copy);
    if (c->s_comp) cudaStreamSynchronize(c->s_comp);
    for (int i = 0; i < N_PUSH_EVENTS; ++i) if (c->push_ev[i]) cudaEventDestroy(c->push_ev[i]);
    for (int i = 0; i < N_DEMOD_EVENTS; ++i) if (c->demod_ev[i].ev) cudaEventDestroy(c->demod_ev[i].ev);
    if (c->tables_ev) cudaEventDestroy(c->tables_ev);
    if (c->own_comp && c->s_comp) cudaStreamDestroy(c->s_comp);
    if (c->own_copy && c->s_copy) cudaStreamDestroy(c->s_copy);
    if (c->own_ws && c->ws) cudaFree(c->ws);
    (void)cudaGetLastError();
    delete c;
}

const char *qld_last_error(const qld_ctx *c) { return c ? c->err.c_str() : g_create_error.c_str(); }

int64_t qld_kernel_launches(const qld_ctx *c) { return c ? c->launches : 0; }

int qld_debug_set_tile(qld_ctx *c, int which, int a, int b, int d)
{
    if (!c) return QLD_E_INVAL;
    if (a < 0 || b < 0 || d < 0) return fail(c, QLD_E_INVAL, "debug_set_tile: negative value");
    if (which == 0) { c->dbg_stream[0] = a; c->dbg_stream[1] = b; }
    else if (which == 1) { c->dbg_tc[0] = a; c->dbg_tc[1] = b; c->dbg_tc[2] = d; c->tmap_valid = false; }
    else if (which == 2 && a <= 2) c->dbg_slide = a;
    else return fail(c, QLD_E_INVAL, "debug_set_tile: which must be 0 (k_demod_stream), 1 (k_demod_tc) or 2 (k_slide_bulk: a = 0 / 1 / 2)");
    return QLD_OK;
}

int qld_accum_mode(const qld_ctx *c) { return c ? c->accum : QLD_E_INVAL; }

const char *qld_last_kernel(const qld_ctx *c) { return (c && c->last_kernel) ? c->last_kernel : ""; }

}  // extern "C"

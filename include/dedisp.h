/*
 * dedisp.h -- C ABI of libdedisp_b200: brute-force incoherent dedispersion on one B200.
 *
 *   out[b][i][t] = sum_{c=0}^{C-1} in[b][c][t + shift(c, dm_i)]            (Algorithm 1)
 *
 * Paper: Sclocco et al., arXiv 1601.01165 ("PAPER.md" below = /root/reference/PAPER.md).
 *   - Algorithm 1 defines the triple loop and `input[chan][sample + Delta]`.
 *   - Eq. (1) defines the delay k = 4150 * DM * (1/f_i^2 - 1/f_h^2) seconds.
 *   - PAPER.md:45 fixes the matrices: input c x t (channel-major), output d x s (DM-major).
 *   - PAPER.md:47 : the delays "can be computed in advance" (the shift table).
 *   - PAPER.md:41, 193 : beams are independent (the nr_beams batch dimension).
 *   - PAPER.md:76 : tunable kernel parameters chosen by auto-tuning (dedisp_tune).
 * Readings of silent/ambiguous points (f_h, operation order, rounding ...): DESIGN.md section 2.
 *
 * Conventions
 *   - Every function returns a dedisp_status (0 = OK); no exception crosses the ABI.
 *   - "device" pointers are CUDA device pointers on the current device; "host" pointers
 *     are ordinary host memory.  The library never frees or keeps caller buffers.
 *   - All work runs in hand-written sm_100a kernels; there is no CPU fallback.
 */
#ifndef DEDISP_B200_H
#define DEDISP_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dedisp_plan dedisp_plan; /* opaque, owned by the library */

typedef enum {
    DEDISP_OK = 0,
    DEDISP_ERR_INVALID_ARG = 1, /* null pointer, non-positive size, negative DM, misalignment */
    DEDISP_ERR_OVERFLOW = 2,    /* a shift, S + M, or a uint8 sum does not fit its integer type */
    DEDISP_ERR_ALLOC = 3,       /* host or device allocation failed */
    DEDISP_ERR_CUDA = 4,        /* CUDA runtime / launch error (no GPU, wrong arch, ...) */
    DEDISP_ERR_IO = 5           /* tuning cache file could not be read / written */
} dedisp_status;

/* in_dtype of dedisp_plan_create */
enum {
    DEDISP_F32 = 0, /* fp32 input, fp32 accumulation and output */
    DEDISP_U8 = 1   /* uint8 input, uint32 output (BASELINE.json config 4; exact) */
};

/* `what` of dedisp_plan_get */
enum {
    DEDISP_MAX_SHIFT = 0,  /* M = max over the table = shift(0, D-1) */
    DEDISP_IN_SAMPLES = 1, /* S + M: samples of each input row that are read (reading A7) */
    DEDISP_IN_PITCH = 2,   /* elements per input row: S + M rounded up to 16 bytes */
    DEDISP_OUT_PITCH = 3,  /* elements per output row = S */
    DEDISP_VARIANT = 4,    /* index of the kernel variant execute() launches */
    DEDISP_NR_CHANNELS = 5,
    DEDISP_NR_DMS = 6,
    DEDISP_NR_SAMPLES = 7,
    DEDISP_IN_DTYPE = 8,
    DEDISP_MAX_STEP = 9,   /* max over (c, i) of shift(c, i+1) - shift(c, i) */
    DEDISP_RESERVED_BEAMS = 10, /* U8 plans: beams the pair workspace holds (dedisp_plan_reserve); else 0 */
    DEDISP_STREAM_H2D_BYTES = 12, /* bytes the last dedisp_stream_block_async call uploaded (0 before the first) */
    DEDISP_PAIR_PITCH = 11 /* U8 plans: 4-byte pairs per row of the pair workspace (nr_samples / 2 rounded up
                              to 4, plus MAX_SHIFT, rounded up to 4): one beam of workspace or static scratch
                              takes nr_channels * PAIR_PITCH * 4 bytes; else 0 */
};

/*
 * dedisp_plan_create -- steps a1-a3 of the path: trial DMs, channel
 * frequencies and the int32 shift table, built ON THE DEVICE in IEEE double with the
 * canonical association (readings A1-A5):
 *     dm_i = dm_first + i*dm_step            f_c = f_low + c*bw      f_h = f_low + C*bw
 *     x    = ((4150*dm_i) * (1/(f_c*f_c) - 1/(f_h*f_h))) * sample_rate          (Eq. 1)
 *     shift(c,i) = floor(x) + (x - floor(x) >= 0.5)
 * Chooses the kernel variant (tuning cache named by $DEDISP_TUNE_CACHE if set, else a
 * heuristic) and prepares it (function attributes, its descriptor table).  nr_samples = S,
 * output samples per beam.  The plan belongs to the CUDA device that is current at creation;
 * every later call on it must be made with the same device current.  A U8 plan whose selected
 * variant is a tree_u8 kernel also allocates the pair workspace for one beam (dedisp_plan_reserve);
 * if there is no memory for it, the plan is created on the best kernel that needs no workspace.
 * Errors: INVALID_ARG (plan == NULL, C/D/S < 1, f_low/bw/rate <= 0 or non-finite,
 * dm_first/dm_step < 0 or non-finite, unknown dtype, or no compiled kernel variant can run the
 * plan); OVERFLOW (shift or S+M > INT32_MAX, or C*255 >= 2^32 for U8); ALLOC; CUDA.  On error
 * *plan = NULL.
 */
int dedisp_plan_create(dedisp_plan **plan, int nr_channels, double f_low_MHz,
                       double channel_bw_MHz, double sample_rate, int64_t nr_samples,
                       double dm_first, double dm_step, int nr_dms, int in_dtype);

/*
 * dedisp_shift_table -- copy Delta(chan, dm) from the DEVICE table the
 * kernels read into caller-owned HOST memory, row-major [nr_dms][nr_channels], int32,
 * entry = shift in samples.  Caller provides nr_dms*nr_channels*4 bytes.
 * Errors: INVALID_ARG (null), CUDA, ALLOC.
 */
int dedisp_shift_table(const dedisp_plan *plan, int32_t *host_out);

/*
 * dedisp_plan_reserve -- U8 plans only (a no-op returning OK for F32 plans): the uint8 register-window
 * kernels read the input through a plan-owned device workspace holding every input row as pairs of
 * samples about S/2 apart (two 16-bit counters per 32-bit add; 4 bytes per pair, C * (S/2 + M) pairs
 * per beam; DEDISP_PAIR_PITCH).  It is allocated for one beam when a tree_u8 variant is first selected
 * (dedisp_plan_create, dedisp_plan_set_variant, dedisp_plan_load_tuning, dedisp_tune, or the first
 * dedisp_execute_variant of such a variant); this call grows it to nr_beams beams so that dedisp_execute
 * runs a whole batch in one kernel launch.  Without it a larger batch still works: dedisp_execute then
 * goes through the workspace as many beams at a time as it holds.
 * Allocates; does not synchronise; never shrinks.  The block it replaces is kept until
 * dedisp_plan_destroy, because kernels in flight and CUDA graphs captured from dedisp_execute earlier
 * still name it: such graphs stay valid (they keep running their old group size), at the price of
 * the old block's memory.  Reserve before the first capture to avoid that.
 * Errors: INVALID_ARG, ALLOC, CUDA.
 */
int dedisp_plan_reserve(dedisp_plan *plan, int nr_beams);

/* dedisp_plan_get -- scalar queries (see the enum).  Errors: INVALID_ARG. */
int dedisp_plan_get(const dedisp_plan *plan, int what, int64_t *value);

/*
 * dedisp_execute -- steps a4-a7: Algorithm 1 for nr_beams beams.
 *   d_in : DEVICE, [nr_beams][nr_channels][IN_PITCH] of float (F32) or uint8_t (U8),
 *          borrowed, read-only, base 16-byte aligned.  Samples [0, S+M) of every row are
 *          read; pitch padding is ignored.  Sample 0 of the input is time-aligned with
 *          output sample 0 at f_h.
 *   d_out: DEVICE, [nr_beams][nr_dms][nr_samples] of float (F32) or uint32_t (U8),
 *          borrowed, fully overwritten, base 16-byte aligned.
 *   stream: a cudaStream_t (NULL = default stream).
 * Asynchronous: enqueues kernels on `stream` and returns; no host sync, no allocation,
 * no host<->device copy, no function-attribute call (all of that happened when the variant
 * was selected), so the first call on a fresh plan can already be captured into a CUDA graph.
 * fp32 sums are accumulated in fp32 in ascending channel order.
 * A plan may be executed repeatedly and concurrently, from several threads and on different streams.
 * F32 calls are independent of each other.  The tree_u8 calls on ONE U8 plan share its pair workspace
 * (dedisp_plan_reserve); the library orders them itself: a call on another stream than the plan's last
 * one makes its stream wait (cudaStreamWaitEvent, no host synchronisation) for that call's kernels, so
 * such calls run one after the other on the GPU instead of overlapping, and every result is correct.
 * One exception: a call made while `stream` is being captured into a CUDA graph neither waits nor is
 * waited for (an event recorded inside a capture cannot order work outside it); replays of such a graph
 * must be ordered by the caller against other calls and replays that use the same U8 plan.
 * Errors: INVALID_ARG (null, nr_beams < 1, misaligned base, current device is not the plan's),
 * CUDA (launch error).
 */
int dedisp_execute(const dedisp_plan *plan, const void *d_in, void *d_out, int nr_beams,
                   void *stream);

/*
 * dedisp_execute_variant -- dedisp_execute with an explicit kernel variant (used by the tuner and the
 * parity tests to drive every compiled variant).  Same contract, except that the first use of a
 * variant on a plan prepares it (one cudaFuncSetAttribute, and for tree variants one descriptor-table
 * allocation and build).  INVALID_ARG if the variant does not support the plan.
 */
int dedisp_execute_variant(const dedisp_plan *plan, int variant, const void *d_in, void *d_out,
                           int nr_beams, void *stream);

/*
 * dedisp_execute_static_scratch -- dedisp_execute for callers that cannot allocate device memory.
 *
 * The uint8 register-window kernels (tree_u8 variants) read the input through a scratch copy in which
 * every row is repacked as pairs of samples (see dedisp_plan_reserve).  dedisp_execute keeps that copy
 * in a plan-owned buffer from cudaMalloc.  Not every caller can have such a buffer: a process whose
 * free device memory already belongs to a pool allocator (PyTorch's caching allocator, RMM) gets
 * "out of memory" from cudaMalloc although the pool has room; a real-time block loop cannot afford
 * cudaMalloc / cudaFree, which serialise the device and stall every other stream; and while another
 * thread captures a CUDA graph in the global capture mode, an allocation call is refused and breaks that
 * capture.  For them this entry point keeps the scratch in a fixed array inside the library image
 * (dedisp_static_scratch_bytes() bytes, 16 MiB; every GPU that loads the library holds that much from
 * load to process exit, used or not).  The call launches kernels and does nothing else: no cudaMalloc,
 * cudaFree, memset, copy, synchronisation or function-attribute call.  The plan itself still comes from
 * dedisp_plan_create, which does allocate (tables, and the workspace this call leaves untouched):
 * create plans in set-up code, before the phase in which allocation is off limits.
 *
 *   plan, d_in, d_out, nr_beams, stream: exactly as for dedisp_execute; same results, bit for bit.
 *   The plan must be a U8 plan whose selected variant (DEDISP_VARIANT) is a tree_u8 kernel; other
 *   plans use no scratch memory and are refused with INVALID_ARG: call dedisp_execute for them.
 *   One beam needs nr_channels * PAIR_PITCH * 4 bytes of scratch (PAIR_PITCH = nr_samples / 2 rounded
 *   up to a multiple of 4, plus MAX_SHIFT, rounded up to 4).  If that exceeds
 *   dedisp_static_scratch_bytes() the call returns INVALID_ARG and dedisp_last_error() names both
 *   sizes.  A batch goes through the array as many beams at a time as fit, in stream order.
 *
 * First call on a device: the library looks up where the array lives on that device
 * (cudaGetSymbolAddress, once per device, with that device current) and remembers it.  Make this first
 * call outside any stream capture; later calls skip the lookup.
 * Sharing: there is ONE array per GPU, shared by every plan, stream and thread of the process, and it
 * keeps what the last call wrote.  No call depends on those contents (each call rewrites every scratch
 * word it later reads, padding included, so nothing needs clearing), but two calls whose kernels can
 * overlap on the GPU (different streams without an event between them) race on the array and
 * produce garbage.  Order all calls of this entry point on one device with respect to each other.
 * It does not touch the plan's own workspace, so it may overlap a dedisp_execute on the same plan.
 * Errors: INVALID_ARG (as dedisp_execute; not a tree_u8 plan; scratch need beyond the maximum;
 * device ordinal >= 64), CUDA (symbol lookup or launch error).
 */
int dedisp_execute_static_scratch(const dedisp_plan *plan, const void *d_in, void *d_out, int nr_beams,
                                  void *stream);

/* Size in bytes of the static scratch array dedisp_execute_static_scratch works in (per GPU). */
int64_t dedisp_static_scratch_bytes(void);

/*
 * dedisp_execute_host -- the same computation for HOST buffers (end-to-end path; the paper keeps
 * data resident on the device, so this is a convenience, not the hot path):
 *   h_in : HOST, [nr_beams][nr_channels][IN_PITCH], borrowed (pinned memory copies fastest);
 *   h_out: HOST, [nr_beams][nr_dms][nr_samples], fully overwritten.
 * Copies h_in to a plan-owned device workspace (allocated or grown on demand, freed by
 * dedisp_plan_destroy), runs dedisp_execute on `stream`, copies the result back and SYNCHRONISES
 * the stream before returning.  Not re-entrant on one plan (the workspace is shared).
 * Errors: INVALID_ARG, ALLOC (workspace), CUDA.
 */
int dedisp_execute_host(dedisp_plan *plan, const void *h_in, void *h_out, int nr_beams,
                        void *stream);

/*
 * dedisp_execute_host_async / dedisp_host_sync -- dedisp_execute_host as a pipeline: the call
 * enqueues H2D copy, kernels and D2H copy on three plan-owned streams over three plan-owned device
 * workspaces (allocated or grown on demand) and returns WITHOUT synchronising, so that consecutive
 * calls overlap the upload of one batch, the kernels of the previous and the download of the one
 * before (the streaming, real-time use the paper targets).  h_in / h_out as in
 * dedisp_execute_host; they must be page-locked for the copies to be asynchronous and must stay
 * valid, and h_in unmodified, until dedisp_host_sync returns (or until three later calls on the
 * plan have been made and synchronised).  Results of call n are complete in h_out after
 * dedisp_host_sync.  Calls on one plan must come from one thread at a time.  dedisp_plan_destroy
 * synchronises and frees the pipeline.
 * Errors: INVALID_ARG, ALLOC (workspaces), CUDA.
 */
int dedisp_execute_host_async(dedisp_plan *plan, const void *h_in, void *h_out, int nr_beams);
int dedisp_host_sync(dedisp_plan *plan);

/*
 * dedisp_stream_block_async -- streaming operation on one beam's long time series (SURVEY.md 8(f)
 * row 4; the paper's real-time setting): dedisperse the block of nr_samples output
 * samples that starts at sample t0, through the same pipeline as dedisp_execute_host_async.
 *   h_series: HOST, [nr_channels][series_pitch] elements; the block needs columns [t0, t0 + S + M) of every row.
 *   h_out   : HOST, [nr_dms][out_pitch] of float / uint32_t; columns [t0, t0 + S) of every row are
 *             written: out[i][t] = sum_c series[c][t + shift(c, dm_i)] for t in the block.
 * Both page-locked and valid until dedisp_host_sync.  The copies are strided (2-D) DMA transfers.
 * Carry-over: consecutive blocks share M input samples per channel.  When a call continues the plan's
 * previous call (same h_series and series_pitch, t0 = previous t0 + S), the shared columns
 * [t0, t0 + M) are NOT uploaded again: they are moved on the device from the previous block's rows, and
 * only the S new columns [t0 + M, t0 + S + M) of every row cross the bus (nr_channels * S elements per
 * block instead of nr_channels * (S + M): 10x fewer for the paper's LOFAR setup, where M = 9 S).  The
 * first block, a block that does not continue the previous one, and the block after dedisp_stream_reset,
 * dedisp_execute_host_async or a workspace growth upload all S + M columns.  Consequence: a change the
 * host makes to columns it has already streamed is not seen by the next block unless dedisp_stream_reset
 * is called first.  dedisp_plan_get(DEDISP_STREAM_H2D_BYTES) tells what the last call uploaded.
 * Errors: INVALID_ARG (null, t0 < 0, series_pitch < t0 + S + M, out_pitch < t0 + S), ALLOC, CUDA.
 */
int dedisp_stream_block_async(dedisp_plan *plan, const void *h_series, int64_t series_pitch,
                              void *h_out, int64_t out_pitch, int64_t t0);

/* dedisp_stream_reset -- forget what the last stream block left on the device: the next
 * dedisp_stream_block_async uploads all S + M columns of its rows.  Enqueues nothing.  Errors: INVALID_ARG. */
int dedisp_stream_reset(dedisp_plan *plan);

/* dedisp_plan_destroy -- frees the plan's host and device tables.  NULL is a no-op. */
int dedisp_plan_destroy(dedisp_plan *plan);

/* ---- kernel variants and the auto-tuner (step a8) ---------- */

/* Number of compiled kernel variants; variants 0 (fp32) and 1 (uint8) are the no-reuse "generic"
 * kernel (one (DM, sample) per thread, global-memory reads: the paper's baseline of PAPER.md:173). */
int dedisp_variant_count(void);

/* Static string "name: DMs/CTA x samples/CTA, outputs/thread, channel-chunk depth ..." or
 * NULL if out of range. */
const char *dedisp_variant_name(int variant);

/* 1 if `variant` can run this plan (dtype, alignment, shared-memory fit), else 0. */
int dedisp_variant_supported(const dedisp_plan *plan, int variant);

/* Select the variant execute() launches and prepare it (function attribute, descriptor table).
 * Errors: INVALID_ARG if unsupported, ALLOC, CUDA. */
int dedisp_plan_set_variant(dedisp_plan *plan, int variant);

/*
 * dedisp_tune -- exhaustive sweep in the spirit of PAPER.md:76 ("try all meaningful
 * combinations and select the best performing one"): times every supported variant on the
 * caller's buffers (same contract as dedisp_execute; d_out is overwritten) with CUDA events
 * on `stream` (synchronises; every variant runs back to back on the one buffer pair the caller gives, so
 * inputs smaller than the 126 MB L2 are timed L2-warm: the kernels are bound on chip, which keeps the
 * ranking, but the absolute times are up to a few per cent below bench.py's, which rotates buffer sets),
 * selects the fastest, and, if cache_path != NULL, persists
 * the winner (one text line "key<TAB>variant name<TAB>note", appended; the last matching line
 * wins on load).  The key is GPU name + setup + a batch-size class (1 beam / 2-7 / 8 or more:
 * the best tile differs when one beam leaves the last wave of CTAs part empty).  ms_out (host, may be NULL)
 * receives variant_count floats: mean ms per call, or -1 for unsupported variants.
 */
int dedisp_tune(dedisp_plan *plan, const void *d_in, void *d_out, int nr_beams, void *stream,
                const char *cache_path, float *ms_out);

/* Load a winner persisted by dedisp_tune for batches of nr_beams beams (the batch-size class of
 * the key; an entry of another class is used if the file has none for this one).  Returns OK and
 * leaves the plan unchanged if the file has no entry for this setup; IO if the file cannot be
 * opened.  *hit (may be NULL) is set to 1 if an entry was applied, else 0. */
int dedisp_plan_load_tuning(dedisp_plan *plan, const char *cache_path, int nr_beams, int *hit);

const char *dedisp_status_string(int status);

/* Last CUDA error text seen by this thread inside the library ("" if none). */
const char *dedisp_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* DEDISP_B200_H */

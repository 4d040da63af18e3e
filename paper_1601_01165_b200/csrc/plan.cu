// plan.cu -- the C-ABI of include/dedisp.h: plan creation (steps a1-a3), queries, execute
// (steps a4-a7) and variant selection.  No CPU fallback exists: every call that needs the device
// fails with DEDISP_ERR_CUDA when there is none.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>

#include "plan_object.h"

namespace dedisp {

static thread_local char g_last_error[256] = "";

void set_last_error(const char *what, cudaError_t e) {
    snprintf(g_last_error, sizeof g_last_error, "%s: %s", what, cudaGetErrorString(e));
}

void set_last_error_text(const char *msg) { snprintf(g_last_error, sizeof g_last_error, "%s", msg); }

#include "build/registry_gen.inc"  // generated from variants.py: kVariantMakers[]

const std::vector<Variant> &variants() {
    static std::vector<Variant> reg;
    static std::once_flag once;
    std::call_once(once, [] {
        for (auto make : kVariantMakers) reg.push_back(make());
    });
    return reg;
}

// Largest shift(c, last DM of tile) - shift(c, first DM of tile) over all channels and DM tiles of
// `dms` DMs: how much longer than the sample tile a staged row can get.
static int span_for(const PlanShape &p, int dms) {
    int span = 0;
    for (int lo = 0; lo < p.D; lo += dms) {
        int hi = std::min(lo + dms - 1, p.D - 1);
        const int32_t *a = p.h_shift + (size_t)lo * p.C, *b = p.h_shift + (size_t)hi * p.C;
        for (int c = 0; c < p.C; ++c) span = std::max(span, b[c] - a[c]);
    }
    return span;
}

static PlanShape shape_of(const dedisp_plan *pl) {
    PlanShape p;
    p.C = pl->C; p.D = pl->D; p.S = (int)pl->S; p.in_pitch = pl->in_pitch; p.dtype = pl->dtype;
    p.M = pl->M; p.max_step = pl->max_step; p.h_shift = pl->h_shift.data(); p.S2 = pl->S2;
    p.tree = &pl->tree;
    return p;
}

static void compute_fits(dedisp_plan *pl) {
    const auto &vs = variants();
    PlanShape p = shape_of(pl);
    std::map<int, int> spans;
    pl->fit.assign(vs.size(), VariantFit());
    for (size_t v = 0; v < vs.size(); ++v) {
        if (vs[v].dtype != pl->dtype) continue;
        int span = 0;
        if (vs[v].kind != KIND_GENERIC) {
            auto it = spans.find(vs[v].dms_cta);
            if (it == spans.end()) it = spans.emplace(vs[v].dms_cta, span_for(p, vs[v].dms_cta)).first;
            span = it->second;
        }
        pl->fit[v] = vs[v].fit(vs[v], p, span);
        pl->fit[v].span = span;
    }
}

// KIND_TREE tables, part 1 (plan creation): per-channel slope classes q_c, kept on the device for the
// descriptor builds.
static cudaError_t build_tree_slopes(dedisp_plan *pl) {
    if (pl->C > 65535) return cudaSuccess;  // grid.y of desc_kernel; such plans use other kinds
    int *d_flags = nullptr;
    int h[2] = {0, 0};
    cudaError_t e;
    if ((e = cudaMalloc(&d_flags, 8)) != cudaSuccess ||
        (e = cudaMalloc(&pl->tree.d_qc, (size_t)pl->C * 4)) != cudaSuccess ||
        (e = cudaMemset(d_flags, 0, 8)) != cudaSuccess ||
        (e = build_chan_slopes(pl->d_shiftT, pl->C, pl->D, pl->dpitch, pl->tree.d_qc, d_flags, 0)) != cudaSuccess ||
        (e = cudaMemcpy(h, d_flags, 8, cudaMemcpyDeviceToHost)) != cudaSuccess)
        set_last_error("build_chan_slopes", e);
    cudaFree(d_flags);
    if (e != cudaSuccess) return e;
    pl->tree.qmax = h[0];
    pl->tree.valid = h[1] == 0;
    return cudaSuccess;
}

// Part 2 (when a tree variant is selected or first run): the descriptor table of the variant's
// (DT, DMs per CTA) pair.  Only the variants that run pay for a table (4 bytes per channel and DM
// group); a failed allocation leaves the plan usable with every other variant.
static int ensure_tree_table(dedisp_plan *pl, int v) {
    const Variant &x = variants()[v];
    if (x.kind != KIND_TREE) return DEDISP_OK;
    std::lock_guard<std::mutex> lk(pl->tree.mu);
    if (pl->tree.find(x.dt, x.dms_cta)) return DEDISP_OK;
    TreeTable t;
    t.dt = x.dt;
    t.dms_cta = x.dms_cta;
    const int nG = (pl->D + x.dt - 1) / x.dt;
    t.pitch = (nG + 31) / 32 * 32 + 32;
    int *d_flags = nullptr;
    int h[2] = {0, 0};
    cudaError_t e;
    if ((e = cudaMalloc(&t.d_desc, (size_t)pl->C * t.pitch * 4)) != cudaSuccess) {
        set_last_error("cudaMalloc(descriptors)", e);
        return DEDISP_ERR_ALLOC;
    }
    if ((e = cudaMalloc(&d_flags, 8)) != cudaSuccess || (e = cudaMemset(d_flags, 0, 8)) != cudaSuccess ||
        (e = build_tree_desc(pl->d_shiftT, pl->tree.d_qc, pl->C, pl->D, pl->dpitch, x.dt, x.dms_cta, 4,
                             t.pitch, t.d_desc, d_flags, 0)) != cudaSuccess ||
        (e = cudaMemcpy(h, d_flags, 8, cudaMemcpyDeviceToHost)) != cudaSuccess) {
        set_last_error("build_tree_desc", e);
        cudaFree(t.d_desc);
        if (d_flags) cudaFree(d_flags);
        return DEDISP_ERR_CUDA;
    }
    cudaFree(d_flags);
    if (h[1] != 0) {  // a window offset past 14 bits: tree_fit excludes such plans
        cudaFree(t.d_desc);
        return DEDISP_ERR_INVALID_ARG;
    }
    pl->tree.tables.push_back(t);
    return DEDISP_OK;
}

// The uint8 tree kernels' pair workspace for nr_beams beams (never shrinks).  An outgrown block is retired,
// not freed: kernels in flight and CUDA graphs captured earlier may still name it, and calls that follow
// are ordered behind the last one by the hand-over event anyway (launch_variant), so no synchronisation is
// needed here.  Retired blocks are freed by dedisp_plan_destroy.
static int grow_pairs(dedisp_plan *pl, int nr_beams) {
    std::lock_guard<std::mutex> lk(pl->pairs_mu);
    if (nr_beams <= pl->pairs_beams) return DEDISP_OK;
    cudaError_t e;
    if (!pl->pairs_done && (e = cudaEventCreateWithFlags(&pl->pairs_done, cudaEventDisableTiming)) != cudaSuccess) {
        set_last_error("cudaEventCreate(pair workspace)", e);
        return DEDISP_ERR_CUDA;
    }
    uint32_t *p = nullptr;
    e = cudaMalloc(&p, (size_t)nr_beams * pl->C * pl->pair_pitch * 4);
    if (e != cudaSuccess) {
        cudaGetLastError();  // the failed allocation must not show up as the next launch's error
        set_last_error("cudaMalloc(pair workspace)", e);
        return DEDISP_ERR_ALLOC;
    }
    try {
        if (pl->d_pairs) pl->retired_pairs.push_back(pl->d_pairs);
    } catch (...) { cudaFree(p); return DEDISP_ERR_ALLOC; }
    pl->d_pairs = p;
    pl->pairs_beams = nr_beams;
    return DEDISP_OK;
}

static bool needs_pairs(const dedisp_plan *pl, int v) {
    return pl->dtype == DEDISP_U8 && variants()[v].kind == KIND_TREE;
}

// Everything a variant needs before its first launch, done when it is SELECTED (plan creation,
// set_variant, load_tuning, tune) so that dedisp_execute itself neither allocates nor touches
// function attributes: the large-shared-memory attribute (per device: set unconditionally, it is
// cheap), for tree variants the descriptor table, and for uint8 tree variants the pair workspace
// (one beam, unless dedisp_plan_reserve asked for more): only the variants that run pay for it.
static int prepare_variant(dedisp_plan *pl, int v) {
    const VariantFit &f = pl->fit[v];
    if (!f.ok) return DEDISP_ERR_INVALID_ARG;
    if (f.smem > 48 * 1024) {
        cudaError_t e = variants()[v].prepare(f.smem);
        if (e != cudaSuccess) { set_last_error("cudaFuncSetAttribute", e); return DEDISP_ERR_CUDA; }
    }
    int rc = ensure_tree_table(pl, v);
    if (rc == DEDISP_OK && needs_pairs(pl, v)) rc = grow_pairs(pl, 1);
    return rc;
}

// Adds per clock and SM the tree tiles sustain on B200 (round-2 measurements on apertif / survey8, tile
// and wave quantisation divided out): {uint8?, DT, samples per thread and DM, warps per CTA, rate}.
// Tiles not listed fall back to a formula.  Only the untuned default uses this; dedisp_tune measures.
static double tree_rate(bool u8, int dt, int tt, int warps, int cc, int lazy) {
    static const struct { int u8, dt, tt, warps; double rate; } kRates[] = {
        {0, 4, 28, 12, 76}, {0, 4, 20, 16, 75}, {0, 5, 20, 12, 74}, {0, 6, 28, 8, 71}, {0, 6, 12, 16, 68}, {0, 4, 20, 12, 66},
        {0, 4, 44, 8, 65},  {0, 5, 12, 16, 63}, {0, 5, 36, 8, 63}, {0, 8, 20, 8, 62},  {0, 6, 12, 12, 60},
        {0, 4, 28, 8, 60},  {0, 4, 12, 16, 60}, {0, 6, 20, 8, 57}, {0, 8, 12, 12, 57}, {0, 4, 36, 8, 62},
        {1, 4, 40, 16, 110}, {1, 5, 24, 16, 108}, {1, 4, 40, 12, 107}, {1, 5, 40, 12, 100}, {1, 4, 24, 16, 101}, {1, 6, 24, 12, 87},
        {1, 6, 24, 16, 84},  {1, 4, 56, 12, 92},  {1, 8, 24, 12, 79},  {1, 4, 72, 8, 82},   {1, 6, 56, 8, 64},
        {1, 8, 40, 8, 47},
    };
    double rate = -1;
    for (const auto &r : kRates)
        if (r.u8 == (int)u8 && r.dt == dt && r.tt == tt && r.warps == warps) rate = r.rate;
    if (rate < 0) {
        const double tile = (double)dt * tt;
        rate = (tile >= 100 ? (warps >= 12 ? 62 : 58) : tile >= 72 ? 52 : 42) * (u8 ? 1.4 : 1.0);
    }
    if (lazy) rate *= u8 ? 1.06 : 1.035;  // upper window quads on demand: ~10 % fewer shared-memory wavefronts
    return rate * (cc >= 12 ? 1.0 : 0.93);  // 8-channel stages: more chunk bookkeeping per add
}

// Untuned default: a cost model in SM clocks.  A CTA costs the larger of its adds at the kind's
// measured rate (adds/clk/SM on B200: tree ~58 for large thread tiles, lds ~28 = the one-word-per-add
// shared-memory cap, generic ~10 = 4-byte loads at the L2's per-SM share; tree tiles: tree_rate) and of the bytes it stages
// from L2 (~40 B/clk/SM); an SM runs ceil(CTAs / SM count of the plan's device) of them (wave quantisation), more slowly when
// too few warps are resident to hide latencies.  dedisp_tune replaces the guess by a measurement.
static int heuristic_variant(const dedisp_plan *pl, bool allow_tree = true) {
    const auto &vs = variants();
    double best = 1e300;
    int bi = -1;  // no variant supports the plan: dedisp_plan_create reports it
    const double esz = pl->dtype == DEDISP_U8 ? 1 : 4;
    for (size_t v = 0; v < vs.size(); ++v) {
        if (!pl->fit[v].ok) continue;
        const Variant &x = vs[v];
        if (!allow_tree && x.kind == KIND_TREE) continue;
        const double tile = (double)x.dt * x.tt;
        double rate, need, occ;
        if (x.kind == KIND_TREE) {
            rate = tree_rate(pl->dtype == DEDISP_U8, x.dt, x.tt, x.threads / 32, x.cc, x.lazy);
            need = 8;
            occ = x.threads <= 128 ? 4 : (x.threads <= 256 && tile <= 48) ? 2 : 1;
        } else if (x.kind == KIND_LDS) {
            rate = (x.dt == 4 && x.tt == 16) ? 30 : tile >= 32 ? 28 : tile >= 16 ? 24 : 14;
            need = 16;
            occ = std::floor(227.0 * 1024 / (double)std::max<size_t>(pl->fit[v].smem, 1));
            occ = std::max(1.0, std::min(occ, std::floor(2048.0 / x.threads)));
        } else {
            rate = 10;
            need = 32;
            occ = 8;
        }
        const double nd = std::ceil((double)pl->D / x.dms_cta), nt = std::ceil((double)pl->S / x.samples_cta);
        const double adds_cta = (double)x.dms_cta * x.samples_cta * pl->C;
        const double bytes_cta = x.kind == KIND_GENERIC ? 0 : (double)pl->C * (x.samples_cta + pl->fit[v].span) * esz;
        const double t_cta = std::max(adds_cta / rate, bytes_cta / 40.0);
        const double n_sm = std::ceil(nd * nt / (double)pl->sm_count);
        const double resident = std::min(occ, n_sm);
        const double warp_eff = std::min(1.0, resident * x.threads / 32.0 / need);
        const double cost = n_sm * t_cta / warp_eff + 6000;  // + launch
        if (cost < best) { best = cost; bi = (int)v; }
    }
    return bi;
}

}  // namespace dedisp

using namespace dedisp;

#define CUDA_TRY(expr, what)              \
    do {                                  \
        cudaError_t e_ = (expr);          \
        if (e_ != cudaSuccess) {          \
            set_last_error(what, e_);     \
            goto cuda_fail;               \
        }                                 \
    } while (0)

extern "C" {

int dedisp_plan_create(dedisp_plan **plan, int nr_channels, double f_low_MHz,
                       double channel_bw_MHz, double sample_rate, int64_t nr_samples,
                       double dm_first, double dm_step, int nr_dms, int in_dtype) {
    if (!plan) return DEDISP_ERR_INVALID_ARG;
    *plan = nullptr;
    auto bad = [](double x) { return !std::isfinite(x); };
    if (nr_channels < 1 || nr_dms < 1 || nr_samples < 1 || bad(f_low_MHz) || bad(channel_bw_MHz) ||
        bad(sample_rate) || bad(dm_first) || bad(dm_step) || f_low_MHz <= 0 || channel_bw_MHz <= 0 ||
        sample_rate <= 0 || dm_first < 0 || dm_step < 0 ||
        (in_dtype != DEDISP_F32 && in_dtype != DEDISP_U8))
        return DEDISP_ERR_INVALID_ARG;
    if (nr_samples > INT32_MAX - 64) return DEDISP_ERR_OVERFLOW;
    if (in_dtype == DEDISP_U8 && (uint64_t)nr_channels * 255u > 0xFFFFFFFFull) return DEDISP_ERR_OVERFLOW;

    dedisp_plan *pl = new (std::nothrow) dedisp_plan();
    if (!pl) return DEDISP_ERR_ALLOC;
    pl->C = nr_channels; pl->D = nr_dms; pl->S = nr_samples; pl->dtype = in_dtype;
    pl->f_low = f_low_MHz; pl->bw = channel_bw_MHz; pl->rate = sample_rate;
    pl->dm_first = dm_first; pl->dm_step = dm_step;
    pl->dpitch = ((nr_dms + 127) / 128) * 128 + 128;
    int *d_flag = nullptr;
    int h_flag = 0;
    int status = DEDISP_ERR_CUDA;
    const int al = in_dtype == DEDISP_U8 ? 16 : 4;
    int64_t in_samples;

    CUDA_TRY(cudaGetDevice(&pl->device), "cudaGetDevice");
    CUDA_TRY(cudaDeviceGetAttribute(&pl->sm_count, cudaDevAttrMultiProcessorCount, pl->device),
             "cudaDeviceGetAttribute(SM count)");
    if (pl->sm_count < 1) pl->sm_count = 1;
    CUDA_TRY(cudaMalloc(&pl->d_shift, (size_t)nr_dms * nr_channels * 4), "cudaMalloc(shift)");
    CUDA_TRY(cudaMalloc(&pl->d_shiftT, (size_t)nr_channels * pl->dpitch * 4), "cudaMalloc(shiftT)");
    CUDA_TRY(cudaMalloc(&d_flag, 4), "cudaMalloc(flag)");
    CUDA_TRY(cudaMemset(d_flag, 0, 4), "cudaMemset");
    CUDA_TRY(build_shift_tables(nr_channels, f_low_MHz, channel_bw_MHz, sample_rate, dm_first,
                                dm_step, nr_dms, pl->dpitch, pl->d_shift, pl->d_shiftT, d_flag, 0),
             "shift_table_kernel");
    CUDA_TRY(cudaMemcpy(&h_flag, d_flag, 4, cudaMemcpyDeviceToHost), "cudaMemcpy(flag)");
    cudaFree(d_flag);
    d_flag = nullptr;
    if (h_flag) { status = DEDISP_ERR_OVERFLOW; goto fail; }
    try {
        pl->h_shift.resize((size_t)nr_dms * nr_channels);
    } catch (...) { status = DEDISP_ERR_ALLOC; goto fail; }
    CUDA_TRY(cudaMemcpy(pl->h_shift.data(), pl->d_shift, pl->h_shift.size() * 4,
                        cudaMemcpyDeviceToHost), "cudaMemcpy(table)");
    pl->M = 0;
    for (int32_t s : pl->h_shift) pl->M = std::max<int64_t>(pl->M, s);
    pl->max_step = 0;
    for (int i = 0; i + 1 < nr_dms; ++i) {
        const int32_t *a = pl->h_shift.data() + (size_t)i * nr_channels, *b = a + nr_channels;
        for (int c = 0; c < nr_channels; ++c) pl->max_step = std::max(pl->max_step, b[c] - a[c]);
    }
    in_samples = nr_samples + pl->M;
    if (in_samples + al > INT32_MAX) { status = DEDISP_ERR_OVERFLOW; goto fail; }
    pl->in_pitch = (int)((in_samples + al - 1) / al * al);
    // uint8 tree kernels: pair y = samples y and y + S2 of a row (kernel_tree.cuh)
    pl->S2 = (int)((((nr_samples + 1) / 2) + 3) & ~(int64_t)3);
    pl->pair_pitch = (int)((pl->S2 + pl->M + 3) & ~(int64_t)3);
    // what the uint8 tree kernels' carry-chain adds rely on (kernel_tree.cuh, gen_tree.py): a register pair
    // (k, k + 1) never straddles the end of the valid pairs, and rows are long enough that what lies past a
    // tile's valid elements only reaches accumulators that are never stored
    if (pl->S2 % 4 != 0 || pl->pair_pitch < pl->S2 + pl->M || pl->pair_pitch % 4 != 0) {
        set_last_error_text("internal: pair layout invariants violated (S2 % 4, pair_pitch >= S2 + M)");
        status = DEDISP_ERR_INVALID_ARG;
        goto fail;
    }
    if (build_tree_slopes(pl) != cudaSuccess) goto cuda_fail;
    compute_fits(pl);
    pl->variant = heuristic_variant(pl);
    if (pl->variant < 0) {
        snprintf(g_last_error, sizeof g_last_error,
                 "no compiled kernel variant supports this plan (nr_dms > 65535 and shifts too long "
                 "for the staged kernels)");
        status = DEDISP_ERR_INVALID_ARG;
        goto fail;
    }
    if (const char *cache = getenv("DEDISP_TUNE_CACHE"))
        if (*cache) dedisp_plan_load_tuning(pl, cache, 1, nullptr);  // missing file / entry: keep the heuristic
    status = prepare_variant(pl, pl->variant);
    if (status == DEDISP_ERR_ALLOC && variants()[pl->variant].kind == KIND_TREE) {
        // no memory for a tree variant's descriptor table or pair workspace: the plan still runs on the
        // best kernel that needs neither
        const int v = heuristic_variant(pl, false);
        if (v >= 0) {
            pl->variant = v;
            status = prepare_variant(pl, v);
        }
    }
    if (status != DEDISP_OK) goto fail;
    *plan = pl;
    return DEDISP_OK;

cuda_fail:
    status = DEDISP_ERR_CUDA;
fail:
    if (d_flag) cudaFree(d_flag);
    dedisp_plan_destroy(pl);
    return status;
}

int dedisp_plan_reserve(dedisp_plan *plan, int nr_beams) {
    if (!plan || nr_beams < 1) return DEDISP_ERR_INVALID_ARG;
    if (plan->dtype != DEDISP_U8 || !plan->tree.valid) return DEDISP_OK;
    return grow_pairs(plan, nr_beams);
}

int dedisp_shift_table(const dedisp_plan *plan, int32_t *host_out) {
    if (!plan || !host_out) return DEDISP_ERR_INVALID_ARG;
    // copied from the DEVICE table the kernels read, not from the host mirror
    cudaError_t e = cudaMemcpy(host_out, plan->d_shift, (size_t)plan->D * plan->C * 4,
                               cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) { set_last_error("cudaMemcpy(table)", e); return DEDISP_ERR_CUDA; }
    return DEDISP_OK;
}

int dedisp_plan_get(const dedisp_plan *plan, int what, int64_t *value) {
    if (!plan || !value) return DEDISP_ERR_INVALID_ARG;
    switch (what) {
        case DEDISP_MAX_SHIFT: *value = plan->M; break;
        case DEDISP_IN_SAMPLES: *value = plan->S + plan->M; break;
        case DEDISP_IN_PITCH: *value = plan->in_pitch; break;
        case DEDISP_OUT_PITCH: *value = plan->S; break;
        case DEDISP_VARIANT: *value = plan->variant; break;
        case DEDISP_NR_CHANNELS: *value = plan->C; break;
        case DEDISP_NR_DMS: *value = plan->D; break;
        case DEDISP_NR_SAMPLES: *value = plan->S; break;
        case DEDISP_IN_DTYPE: *value = plan->dtype; break;
        case DEDISP_MAX_STEP: *value = plan->max_step; break;
        case DEDISP_RESERVED_BEAMS: *value = plan->dtype == DEDISP_U8 ? plan->pairs_beams : 0; break;
        case DEDISP_PAIR_PITCH: *value = plan->dtype == DEDISP_U8 ? plan->pair_pitch : 0; break;
        case DEDISP_STREAM_H2D_BYTES: *value = plan->pipe.st_h2d_bytes; break;
        default: return DEDISP_ERR_INVALID_ARG;
    }
    return DEDISP_OK;
}

// Enqueue variant v for nr_beams beams.  Kernels only: no allocation, no host synchronisation.
static int launch_variant(const dedisp_plan *plan, int v, const void *d_in, void *d_out,
                          int nr_beams, cudaStream_t st) {
    const Variant &x = variants()[v];
    const VariantFit &f = plan->fit[v];
    KArgs a;
    a.in = d_in; a.out = d_out; a.shift = plan->d_shift; a.shiftT = plan->d_shiftT;
    a.C = plan->C; a.D = plan->D; a.S = (int)plan->S; a.in_pitch = plan->in_pitch;
    a.dpitch = plan->dpitch; a.lrow = f.lrow;
    a.pairs = plan->d_pairs; a.pair_pitch = plan->pair_pitch; a.S2 = plan->S2;
    const TreeTable *tt = x.kind == KIND_TREE ? plan->tree.find_locked(x.dt, x.dms_cta) : nullptr;
    if (x.kind == KIND_TREE && !tt) return DEDISP_ERR_INVALID_ARG;  // variant was never prepared
    a.desc = tt ? tt->d_desc : nullptr;
    a.descpitch = tt ? tt->pitch : 0;
    // grid.z carries the beams (step a7): at most 65535 per launch; the uint8 tree kernels
    // go through the pair workspace, as many beams at a time as it was reserved for
    const bool paired = x.kind == KIND_TREE && plan->dtype == DEDISP_U8;
    // Paired calls on one plan share its pair workspace.  The whole enqueue happens under the plan's
    // workspace mutex, and the workspace is handed from stream to stream by an event: a call on another
    // stream than the last paired call's first makes its stream wait for that call's kernels, so calls on
    // different streams (or from different threads) never overlap on the workspace, whatever the caller
    // does.  No host synchronisation.  Not while `st` is being captured: events recorded in a capture
    // cannot order work outside it, so a captured call neither waits nor records, and replays of the graph
    // are for the caller to order against other calls on the plan (include/dedisp.h).
    std::unique_lock<std::mutex> pairs_lock(plan->pairs_mu, std::defer_lock);
    bool hand_over = false;
    if (paired) {
        pairs_lock.lock();
        if (!plan->d_pairs || plan->pairs_beams < 1) return DEDISP_ERR_INVALID_ARG;
        a.pairs = plan->d_pairs;
        cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(st, &cap) != cudaSuccess) { cudaGetLastError(); cap = cudaStreamCaptureStatusNone; }
        hand_over = cap == cudaStreamCaptureStatusNone;
        if (hand_over && plan->pairs_used && plan->pairs_stream != st) {
            cudaError_t e = cudaStreamWaitEvent(st, plan->pairs_done, 0);
            if (e != cudaSuccess) { set_last_error("cudaStreamWaitEvent(pair workspace)", e); return DEDISP_ERR_CUDA; }
        }
    }
    const int group = paired ? std::min(plan->pairs_beams, 65535) : 65535;
    const size_t in_beam = (size_t)plan->C * plan->in_pitch * (plan->dtype == DEDISP_U8 ? 1 : 4);
    const size_t out_beam = (size_t)plan->D * plan->S * 4;
    for (int b0 = 0; b0 < nr_beams; b0 += group) {
        int nb = std::min(group, nr_beams - b0);
        a.in = (const char *)d_in + (size_t)b0 * in_beam;
        a.out = (char *)d_out + (size_t)b0 * out_beam;
        cudaError_t e = cudaSuccess;
        if (paired)
            e = pack_pairs((const uint8_t *)a.in, plan->d_pairs, nb, plan->C, plan->in_pitch,
                           plan->pair_pitch, plan->S2, st);
        if (e == cudaSuccess) e = x.launch(a, nb, f.smem, st);
        if (e != cudaSuccess) { set_last_error(x.name, e); return DEDISP_ERR_CUDA; }
    }
    if (hand_over) {
        cudaError_t e = cudaEventRecord(plan->pairs_done, st);
        if (e != cudaSuccess) { set_last_error("cudaEventRecord(pair workspace)", e); return DEDISP_ERR_CUDA; }
        plan->pairs_stream = st;
        plan->pairs_used = true;
    }
    return DEDISP_OK;
}

static int check_execute_args(const dedisp_plan *plan, const void *d_in, void *d_out, int nr_beams) {
    if (!plan || !d_in || !d_out || nr_beams < 1) return DEDISP_ERR_INVALID_ARG;
    if (((uintptr_t)d_in & 15) || ((uintptr_t)d_out & 15)) return DEDISP_ERR_INVALID_ARG;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != plan->device) {
        snprintf(g_last_error, sizeof g_last_error,
                 "the plan lives on device %d but the current device is %d", plan->device, dev);
        return DEDISP_ERR_INVALID_ARG;
    }
    return DEDISP_OK;
}

int dedisp_execute_variant(const dedisp_plan *plan, int variant, const void *d_in, void *d_out,
                           int nr_beams, void *stream) {
    int rc = check_execute_args(plan, d_in, d_out, nr_beams);
    if (rc != DEDISP_OK) return rc;
    if (variant < 0 || variant >= (int)variants().size() || !plan->fit[variant].ok)
        return DEDISP_ERR_INVALID_ARG;
    // an explicitly chosen variant may not have been selected before: prepare it here (this is the
    // tuner's and the tests' entry point; dedisp_execute never takes this branch's allocations)
    rc = prepare_variant(const_cast<dedisp_plan *>(plan), variant);
    if (rc != DEDISP_OK) return rc;
    return launch_variant(plan, variant, d_in, d_out, nr_beams, (cudaStream_t)stream);
}

int dedisp_execute(const dedisp_plan *plan, const void *d_in, void *d_out, int nr_beams,
                   void *stream) {
    int rc = check_execute_args(plan, d_in, d_out, nr_beams);
    if (rc != DEDISP_OK) return rc;
    return launch_variant(plan, plan->variant, d_in, d_out, nr_beams, (cudaStream_t)stream);
}

int dedisp_execute_host(dedisp_plan *plan, const void *h_in, void *h_out, int nr_beams,
                        void *stream) {
    if (!plan || !h_in || !h_out || nr_beams < 1) return DEDISP_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t in_bytes = (size_t)nr_beams * plan->C * plan->in_pitch * (plan->dtype == DEDISP_U8 ? 1 : 4);
    const size_t out_bytes = (size_t)nr_beams * plan->D * plan->S * 4;
    cudaError_t e;
    if (plan->ws_in_bytes < in_bytes) {
        if (plan->ws_in) cudaFree(plan->ws_in);
        plan->ws_in = nullptr; plan->ws_in_bytes = 0;
        e = cudaMalloc(&plan->ws_in, in_bytes);
        if (e != cudaSuccess) { set_last_error("cudaMalloc(ws_in)", e); return DEDISP_ERR_ALLOC; }
        plan->ws_in_bytes = in_bytes;
    }
    if (plan->ws_out_bytes < out_bytes) {
        if (plan->ws_out) cudaFree(plan->ws_out);
        plan->ws_out = nullptr; plan->ws_out_bytes = 0;
        e = cudaMalloc(&plan->ws_out, out_bytes);
        if (e != cudaSuccess) { set_last_error("cudaMalloc(ws_out)", e); return DEDISP_ERR_ALLOC; }
        plan->ws_out_bytes = out_bytes;
    }
    e = cudaMemcpyAsync(plan->ws_in, h_in, in_bytes, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) { set_last_error("cudaMemcpyAsync(H2D)", e); return DEDISP_ERR_CUDA; }
    int rc = dedisp_execute(plan, plan->ws_in, plan->ws_out, nr_beams, stream);
    if (rc != DEDISP_OK) return rc;
    e = cudaMemcpyAsync(h_out, plan->ws_out, out_bytes, cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) { set_last_error("cudaMemcpyAsync(D2H)", e); return DEDISP_ERR_CUDA; }
    e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { set_last_error("cudaStreamSynchronize", e); return DEDISP_ERR_CUDA; }
    return DEDISP_OK;
}

int dedisp_plan_destroy(dedisp_plan *plan) {
    if (!plan) return DEDISP_OK;
    plan->pipe.destroy();  // drains the host pipeline's streams first
    if (plan->d_shift) cudaFree(plan->d_shift);
    if (plan->d_shiftT) cudaFree(plan->d_shiftT);
    if (plan->tree.d_qc) cudaFree(plan->tree.d_qc);
    for (auto &t : plan->tree.tables)
        if (t.d_desc) cudaFree(t.d_desc);
    if (plan->d_pairs) cudaFree(plan->d_pairs);
    for (uint32_t *p : plan->retired_pairs) cudaFree(p);
    if (plan->pairs_done) cudaEventDestroy(plan->pairs_done);
    if (plan->ws_in) cudaFree(plan->ws_in);
    if (plan->ws_out) cudaFree(plan->ws_out);
    delete plan;
    return DEDISP_OK;
}

int dedisp_variant_count(void) { return (int)variants().size(); }

const char *dedisp_variant_name(int variant) {
    if (variant < 0 || variant >= (int)variants().size()) return nullptr;
    return variants()[variant].name;
}

int dedisp_variant_supported(const dedisp_plan *plan, int variant) {
    if (!plan || variant < 0 || variant >= (int)variants().size()) return 0;
    return plan->fit[variant].ok ? 1 : 0;
}

int dedisp_plan_set_variant(dedisp_plan *plan, int variant) {
    if (!dedisp_variant_supported(plan, variant)) return DEDISP_ERR_INVALID_ARG;
    int rc = prepare_variant(plan, variant);
    if (rc != DEDISP_OK) return rc;
    plan->variant = variant;
    return DEDISP_OK;
}

const char *dedisp_status_string(int status) {
    switch (status) {
        case DEDISP_OK: return "ok";
        case DEDISP_ERR_INVALID_ARG: return "invalid argument";
        case DEDISP_ERR_OVERFLOW: return "integer overflow";
        case DEDISP_ERR_ALLOC: return "allocation failed";
        case DEDISP_ERR_CUDA: return "CUDA error";
        case DEDISP_ERR_IO: return "tuning cache I/O error";
        default: return "unknown status";
    }
}

const char *dedisp_last_error(void) { return g_last_error; }

}  // extern "C"

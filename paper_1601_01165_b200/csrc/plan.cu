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

#include "dedisp_internal.h"

namespace dedisp {

static thread_local char g_last_error[256] = "";

void set_last_error(const char *what, cudaError_t e) {
    snprintf(g_last_error, sizeof g_last_error, "%s: %s", what, cudaGetErrorString(e));
}

// one per row of TREE_VARIANTS in variants_tree.cu
void register_tree0(std::vector<Variant> &);
void register_tree1(std::vector<Variant> &);
void register_tree2(std::vector<Variant> &);
void register_tree3(std::vector<Variant> &);
void register_tree4(std::vector<Variant> &);
void register_tree5(std::vector<Variant> &);
void register_tree6(std::vector<Variant> &);
void register_tree7(std::vector<Variant> &);
void register_tree8(std::vector<Variant> &);
void register_tree9(std::vector<Variant> &);
void register_tree10(std::vector<Variant> &);
void register_tree11(std::vector<Variant> &);
void register_tree12(std::vector<Variant> &);
void register_tree13(std::vector<Variant> &);
void register_tree14(std::vector<Variant> &);
void register_tree15(std::vector<Variant> &);
void register_tree16(std::vector<Variant> &);
void register_tree17(std::vector<Variant> &);
void register_tree18(std::vector<Variant> &);
void register_tree19(std::vector<Variant> &);
void register_tree20(std::vector<Variant> &);
void register_tree21(std::vector<Variant> &);
void register_tree22(std::vector<Variant> &);
void register_tree23(std::vector<Variant> &);
void register_tree24(std::vector<Variant> &);
void register_tree25(std::vector<Variant> &);
void register_tree26(std::vector<Variant> &);
void register_tree27(std::vector<Variant> &);
void register_tree28(std::vector<Variant> &);
void register_tree29(std::vector<Variant> &);
void register_tree30(std::vector<Variant> &);
void register_tree31(std::vector<Variant> &);
void register_tree(std::vector<Variant> &r) {
    void (*parts[])(std::vector<Variant> &) = {
        register_tree0, register_tree1, register_tree2, register_tree3, register_tree4, register_tree5, register_tree6, register_tree7, register_tree8, register_tree9, register_tree10, register_tree11, register_tree12, register_tree13, register_tree14, register_tree15, register_tree16, register_tree17, register_tree18, register_tree19,
        register_tree20, register_tree21, register_tree22, register_tree23, register_tree24,
        register_tree25, register_tree26, register_tree27, register_tree28, register_tree29, register_tree30, register_tree31};
    for (auto f : parts) f(r);
}

const std::vector<Variant> &variants() {
    static std::vector<Variant> reg;
    static std::once_flag once;
    std::call_once(once, [] {
        register_generic(reg);  // variants 0 (f32) and 1 (u8): the no-reuse baseline
        register_lds(reg);
        register_u8(reg);
        register_tree(reg);
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
    p.M = pl->M; p.max_step = pl->max_step; p.h_shift = pl->h_shift.data();
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

// KIND_TREE tables: per-channel slope classes, then one descriptor table per (DT, DMs per CTA)
// pair some registered variant uses.
static cudaError_t build_tree_tables(dedisp_plan *pl) {
    if (pl->C > 65535) return cudaSuccess;  // grid.y of desc_kernel; such plans use other kinds
    int *d_flags = nullptr, *d_qc = nullptr;
    int h[2] = {0, 0};
    cudaError_t e;
    if ((e = cudaMalloc(&d_flags, 8)) != cudaSuccess || (e = cudaMalloc(&d_qc, (size_t)pl->C * 4)) != cudaSuccess ||
        (e = cudaMemset(d_flags, 0, 8)) != cudaSuccess ||
        (e = build_chan_slopes(pl->d_shiftT, pl->C, pl->D, pl->dpitch, d_qc, d_flags, 0)) != cudaSuccess ||
        (e = cudaMemcpy(h, d_flags, 8, cudaMemcpyDeviceToHost)) != cudaSuccess) {
        set_last_error("build_chan_slopes", e);
        cudaFree(d_flags);
        cudaFree(d_qc);
        return e;
    }
    pl->tree.qmax = h[0];
    pl->tree.valid = h[1] == 0;
    if (pl->tree.valid) {
        for (const Variant &v : variants()) {
            if (v.kind != KIND_TREE || v.dtype != pl->dtype || v.rstep < pl->tree.qmax) continue;
            if (pl->tree.find(v.dt, v.dms_cta)) continue;
            TreeTable t;
            t.dt = v.dt;
            t.dms_cta = v.dms_cta;
            const int nG = (pl->D + v.dt - 1) / v.dt;
            t.pitch = (nG + 31) / 32 * 32 + 32;
            if ((e = cudaMalloc(&t.d_desc, (size_t)pl->C * t.pitch * 4)) != cudaSuccess) break;
            pl->tree.tables.push_back(t);  // owned by the plan from here on
            if ((e = cudaMemset(d_flags, 0, 8)) != cudaSuccess ||
                (e = build_tree_desc(pl->d_shiftT, d_qc, pl->C, pl->D, pl->dpitch, v.dt, v.dms_cta,
                                     pl->dtype == DEDISP_U8 ? 16 : 4, t.pitch, t.d_desc, d_flags,
                                     0)) != cudaSuccess ||
                (e = cudaMemcpy(h, d_flags, 8, cudaMemcpyDeviceToHost)) != cudaSuccess)
                break;
            pl->tree.tables.back().valid = h[1] == 0;
        }
        if (e != cudaSuccess) set_last_error("build_tree_desc", e);
    }
    cudaFree(d_flags);
    cudaFree(d_qc);
    return e;
}

// Untuned default: a cost model in SM clocks.  A CTA costs the larger of its adds at the kind's
// measured rate (adds/clk/SM on B200: tree ~58 for large thread tiles, lds ~28 = the one-word-per-add
// shared-memory cap, generic ~10 = 4-byte loads at the L2's per-SM share) and of the bytes it stages
// from L2 (~40 B/clk/SM); an SM runs ceil(CTAs / 148) of them (wave quantisation), more slowly when
// too few warps are resident to hide latencies.  dedisp_tune replaces the guess by a measurement.
static int heuristic_variant(const dedisp_plan *pl) {
    const auto &vs = variants();
    double best = 1e300;
    int bi = pl->dtype == DEDISP_U8 ? 1 : 0;
    const double esz = pl->dtype == DEDISP_U8 ? 1 : 4;
    for (size_t v = 0; v < vs.size(); ++v) {
        if (!pl->fit[v].ok) continue;
        const Variant &x = vs[v];
        const double tile = (double)x.dt * x.tt;
        double rate, need, occ;
        if (x.kind == KIND_TREE) {
            rate = (tile >= 100 ? (x.threads >= 384 ? 62 : 58) : tile >= 72 ? 52 : 42) *
                   (pl->dtype == DEDISP_U8 ? 0.85 : 1.0);
            need = 8;
            occ = x.threads <= 128 ? 4 : (x.threads <= 256 && tile <= 48) ? 2 : 1;
        } else if (x.kind == KIND_LDS) {
            rate = tile >= 32 ? 28 : tile >= 16 ? 24 : 14;
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
        const double n_sm = std::ceil(nd * nt / 148.0);
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
    if (build_tree_tables(pl) != cudaSuccess) goto cuda_fail;
    compute_fits(pl);
    pl->variant = heuristic_variant(pl);
    if (const char *cache = getenv("DEDISP_TUNE_CACHE"))
        if (*cache) dedisp_plan_load_tuning(pl, cache);  // missing file / entry: keep the heuristic
    *plan = pl;
    return DEDISP_OK;

cuda_fail:
    status = DEDISP_ERR_CUDA;
fail:
    if (d_flag) cudaFree(d_flag);
    dedisp_plan_destroy(pl);
    return status;
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
        default: return DEDISP_ERR_INVALID_ARG;
    }
    return DEDISP_OK;
}

static int launch_variant(const dedisp_plan *plan, int v, const void *d_in, void *d_out,
                          int nr_beams, cudaStream_t st) {
    const Variant &x = variants()[v];
    const VariantFit &f = plan->fit[v];
    KArgs a;
    a.in = d_in; a.out = d_out; a.shift = plan->d_shift; a.shiftT = plan->d_shiftT;
    a.C = plan->C; a.D = plan->D; a.S = (int)plan->S; a.in_pitch = plan->in_pitch;
    a.dpitch = plan->dpitch; a.lrow = f.lrow;
    const TreeTable *tt = x.kind == KIND_TREE ? plan->tree.find(x.dt, x.dms_cta) : nullptr;
    a.desc = tt ? tt->d_desc : nullptr;
    a.descpitch = tt ? tt->pitch : 0;
    // grid.z carries the beams (step a7): at most 65535 per launch
    const size_t in_beam = (size_t)plan->C * plan->in_pitch * (plan->dtype == DEDISP_U8 ? 1 : 4);
    const size_t out_beam = (size_t)plan->D * plan->S * 4;
    for (int b0 = 0; b0 < nr_beams; b0 += 65535) {
        int nb = std::min(65535, nr_beams - b0);
        a.in = (const char *)d_in + (size_t)b0 * in_beam;
        a.out = (char *)d_out + (size_t)b0 * out_beam;
        cudaError_t e = x.launch(a, nb, f.smem, st);
        if (e != cudaSuccess) { set_last_error(x.name, e); return DEDISP_ERR_CUDA; }
    }
    return DEDISP_OK;
}

// cudaFuncSetAttribute once per (variant, device context); cheap to repeat, so no global state
// beyond a per-process flag array.
static int prepare_variant(const dedisp_plan *plan, int v) {
    static std::mutex mu;
    static std::vector<size_t> prepared;
    std::lock_guard<std::mutex> lk(mu);
    if (prepared.size() != variants().size()) prepared.assign(variants().size(), 0);
    size_t need = plan->fit[v].smem;
    if (need <= prepared[v] || need <= 48 * 1024) return DEDISP_OK;
    cudaError_t e = variants()[v].prepare(need);
    if (e != cudaSuccess) { set_last_error("cudaFuncSetAttribute", e); return DEDISP_ERR_CUDA; }
    prepared[v] = need;
    return DEDISP_OK;
}

int dedisp_execute_variant(const dedisp_plan *plan, int variant, const void *d_in, void *d_out,
                           int nr_beams, void *stream) {
    if (!plan || !d_in || !d_out || nr_beams < 1) return DEDISP_ERR_INVALID_ARG;
    if (((uintptr_t)d_in & 15) || ((uintptr_t)d_out & 15)) return DEDISP_ERR_INVALID_ARG;
    if (variant < 0 || variant >= (int)variants().size() || !plan->fit[variant].ok)
        return DEDISP_ERR_INVALID_ARG;
    int rc = prepare_variant(plan, variant);
    if (rc != DEDISP_OK) return rc;
    return launch_variant(plan, variant, d_in, d_out, nr_beams, (cudaStream_t)stream);
}

int dedisp_execute(const dedisp_plan *plan, const void *d_in, void *d_out, int nr_beams,
                   void *stream) {
    if (!plan) return DEDISP_ERR_INVALID_ARG;
    return dedisp_execute_variant(plan, plan->variant, d_in, d_out, nr_beams, stream);
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
    if (plan->d_shift) cudaFree(plan->d_shift);
    if (plan->d_shiftT) cudaFree(plan->d_shiftT);
    for (auto &t : plan->tree.tables)
        if (t.d_desc) cudaFree(t.d_desc);
    if (plan->ws_in) cudaFree(plan->ws_in);
    if (plan->ws_out) cudaFree(plan->ws_out);
    plan->pipe.destroy();
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

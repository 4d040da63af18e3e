// tuner.cu -- step a8: the auto-tuner ("try all meaningful combinations and select the
// best performing one"; the optimum differs per observational setup).  Sweeps the
// compiled variants (DMs/CTA x samples/CTA x outputs/thread x channel-chunk depth), times each with
// CUDA events on the caller's stream, and persists the winner per (GPU, setup, batch class) as one
// text line.
#include <cstdio>
#include <cstring>
#include <fstream>
#include <sstream>
#include <string>

#include "plan_object.h"

using namespace dedisp;

// 1 beam / 2-7 / >= 8: one beam leaves the last wave of CTAs part empty, a large batch does not, so
// their winners can differ.
static int beams_class(int nr_beams) { return nr_beams <= 1 ? 1 : nr_beams < 8 ? 2 : 8; }

static std::string setup_key(const dedisp_plan *pl, int bclass) {
    cudaDeviceProp prop;
    char gpu[256] = "unknown";
    if (cudaGetDeviceProperties(&prop, pl->device) == cudaSuccess)
        snprintf(gpu, sizeof gpu, "%s", prop.name);
    char buf[640];
    snprintf(buf, sizeof buf,
             "gpu=%s;C=%d;f_low=%.17g;bw=%.17g;rate=%.17g;S=%lld;dm_first=%.17g;dm_step=%.17g;D=%d;"
             "dtype=%d;beams=%d",
             gpu, pl->C, pl->f_low, pl->bw, pl->rate, (long long)pl->S, pl->dm_first, pl->dm_step,
             pl->D, pl->dtype, bclass);
    return buf;
}

extern "C" int dedisp_plan_load_tuning(dedisp_plan *plan, const char *cache_path, int nr_beams,
                                       int *hit) {
    if (hit) *hit = 0;
    if (!plan || !cache_path || nr_beams < 1) return DEDISP_ERR_INVALID_ARG;
    std::ifstream f(cache_path);
    if (!f) return DEDISP_ERR_IO;
    // the wanted batch class first, then the others as a fallback
    const int want = beams_class(nr_beams);
    const int order[3] = {want, want == 8 ? 2 : 8, want == 1 ? 2 : 1};
    std::string winners[3];
    std::string keys[3];
    for (int i = 0; i < 3; ++i) keys[i] = setup_key(plan, order[i]);
    std::string line;
    while (std::getline(f, line)) {
        size_t tab = line.find('\t');
        if (tab == std::string::npos) continue;
        for (int i = 0; i < 3; ++i)
            if (line.compare(0, tab, keys[i]) == 0) {
                size_t tab2 = line.find('\t', tab + 1);
                winners[i] = line.substr(tab + 1, tab2 == std::string::npos ? std::string::npos
                                                                            : tab2 - tab - 1);  // last entry wins
            }
    }
    const auto &vs = variants();
    for (int i = 0; i < 3; ++i) {
        if (winners[i].empty()) continue;
        for (size_t v = 0; v < vs.size(); ++v)
            if (winners[i] == vs[v].name && plan->fit[v].ok) {
                int rc = dedisp_plan_set_variant(plan, (int)v);
                if (rc != DEDISP_OK) return rc;
                if (hit) *hit = 1;
                return DEDISP_OK;
            }
    }
    return DEDISP_OK;
}

extern "C" int dedisp_tune(dedisp_plan *plan, const void *d_in, void *d_out, int nr_beams,
                           void *stream, const char *cache_path, float *ms_out) {
    if (!plan || !d_in || !d_out || nr_beams < 1) return DEDISP_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const auto &vs = variants();
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        set_last_error("cudaEventCreate", cudaGetLastError());
        return DEDISP_ERR_CUDA;
    }
    int best = -1;
    float best_ms = 0.f;
    int rc = DEDISP_OK;
    for (size_t v = 0; v < vs.size(); ++v) {
        if (ms_out) ms_out[v] = -1.f;
        if (!plan->fit[v].ok) continue;
        // one warm-up (also prepares the variant), then a timed batch sized from a single call
        rc = dedisp_execute_variant(plan, (int)v, d_in, d_out, nr_beams, stream);
        if (rc == DEDISP_ERR_ALLOC) { rc = DEDISP_OK; continue; }  // no room for its table: skip it
        if (rc != DEDISP_OK) break;
        cudaEventRecord(e0, st);
        rc = dedisp_execute_variant(plan, (int)v, d_in, d_out, nr_beams, stream);
        cudaEventRecord(e1, st);
        cudaError_t e = cudaEventSynchronize(e1);
        if (rc != DEDISP_OK) break;
        if (e != cudaSuccess) { set_last_error(vs[v].name, e); rc = DEDISP_ERR_CUDA; break; }
        float ms1 = 0.f;
        cudaEventElapsedTime(&ms1, e0, e1);
        // skip the long batch for variants already 3x slower than the best
        float ms = ms1;
        if (best < 0 || ms1 < 3.f * best_ms) {
            int reps = ms1 > 0.f ? (int)(30.f / ms1) : 10;  // about 30 ms per variant
            reps = reps < 3 ? 3 : reps > 50 ? 50 : reps;
            cudaEventRecord(e0, st);
            for (int r = 0; r < reps && rc == DEDISP_OK; ++r)
                rc = dedisp_execute_variant(plan, (int)v, d_in, d_out, nr_beams, stream);
            cudaEventRecord(e1, st);
            e = cudaEventSynchronize(e1);
            if (rc != DEDISP_OK) break;
            if (e != cudaSuccess) { set_last_error(vs[v].name, e); rc = DEDISP_ERR_CUDA; break; }
            cudaEventElapsedTime(&ms, e0, e1);
            ms /= reps;
        }
        if (ms_out) ms_out[v] = ms;
        if (best < 0 || ms < best_ms) { best = (int)v; best_ms = ms; }
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (rc != DEDISP_OK) return rc;
    if (best < 0) return DEDISP_ERR_INVALID_ARG;
    rc = dedisp_plan_set_variant(plan, best);
    if (rc != DEDISP_OK) return rc;
    if (cache_path) {
        FILE *f = fopen(cache_path, "a");
        if (!f) return DEDISP_ERR_IO;
        fprintf(f, "%s\t%s\t%.6f ms, %d beams\n", setup_key(plan, beams_class(nr_beams)).c_str(),
                vs[best].name, best_ms, nr_beams);
        if (fclose(f) != 0) return DEDISP_ERR_IO;
    }
    return DEDISP_OK;
}

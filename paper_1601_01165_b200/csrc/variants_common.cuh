// variants_common.cuh -- turns a Tile<> instantiation into a registry entry (step a8: the set of
// tunable configurations the auto-tuner sweeps).
#pragma once
#include <cstdio>

#include "kernels.cuh"

namespace dedisp {

constexpr size_t kMaxSmem = 227 * 1024;

template <typename T>
VariantFit tiled_fit(const Variant &v, const PlanShape &p, int span_cta) {
    VariantFit f;
    if (p.dtype != v.dtype) return f;
    long lrow = (long)T::SAMPLES_CTA + span_cta + 2 * T::AL + 0;
    lrow = (lrow + T::AL - 1) / T::AL * T::AL;
    size_t smem = tile_smem_bytes<T>((int)lrow);
    if (smem > kMaxSmem) return f;
    if ((p.S + T::SAMPLES_CTA - 1) / T::SAMPLES_CTA > 65535) return f;
    f.ok = true;
    f.lrow = (int)lrow;
    f.smem = smem;
    return f;
}

template <typename T>
cudaError_t tiled_launch(const KArgs &a, int nr_beams, size_t smem, cudaStream_t st) {
    dim3 grid((a.D + T::DMS_CTA - 1) / T::DMS_CTA, (a.S + T::SAMPLES_CTA - 1) / T::SAMPLES_CTA,
              nr_beams);
    tiled_kernel<T><<<grid, T::THREADS, smem, st>>>(a);
    return cudaGetLastError();
}

template <typename T>
cudaError_t tiled_prepare(size_t smem) {
    return cudaFuncSetAttribute(tiled_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)smem);
}

// name: "lds_<dtype>: DMSxSAMPLES DMsxsamples/CTA, dtxtt outputs/thread, ccN sN bN" (static storage).
template <typename T>
Variant make_tiled() {
    static char name[96];
    const char *dt = sizeof(typename T::In) == 1 ? "u8" : "f32";
    snprintf(name, sizeof name, "lds_%s: %dx%d DMsxsamples/CTA, %dx%d outputs/thread, cc%d s%d b%d", dt,
             T::DMS_CTA, T::SAMPLES_CTA, T::DT, T::TT, T::CC, T::NSTAGE, T::MINB);
    Variant v;
    v.name = name;
    v.dtype = sizeof(typename T::In) == 1 ? DEDISP_U8 : DEDISP_F32;
    v.kind = T::KIND;
    v.dms_cta = T::DMS_CTA;
    v.samples_cta = T::SAMPLES_CTA;
    v.dt = T::DT;
    v.tt = T::TT;
    v.cc = T::CC;
    v.stages = T::NSTAGE;
    v.rstep = 0;
    v.threads = T::THREADS;
    v.fit = tiled_fit<T>;
    v.launch = tiled_launch<T>;
    v.prepare = tiled_prepare<T>;
    return v;
}

}  // namespace dedisp

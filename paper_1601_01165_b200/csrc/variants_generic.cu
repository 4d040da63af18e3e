// variants_generic.cu -- variant 0/1: the no-reuse kernel.
#include "variants_common.cuh"

namespace dedisp {

template <typename In>
static VariantFit generic_fit(const Variant &v, const PlanShape &p, int) {
    VariantFit f;
    f.ok = p.dtype == v.dtype && p.D <= 65535;
    return f;
}
template <typename In>
static cudaError_t generic_launch(const KArgs &a, int nr_beams, size_t, cudaStream_t st) {
    dim3 grid((a.S + 255) / 256, a.D, nr_beams);
    generic_kernel<In><<<grid, 256, 0, st>>>(a);
    return cudaGetLastError();
}
static cudaError_t no_prepare(size_t) { return cudaSuccess; }

template <typename In>
static Variant make_generic(const char *name, int dtype) {
    Variant v;
    v.name = name;
    v.dtype = dtype;
    v.kind = KIND_GENERIC;
    v.dms_cta = 1;
    v.samples_cta = 256;
    v.dt = v.tt = 1;
    v.cc = 0;
    v.stages = 0;
    v.rstep = 0;
    v.threads = 256;
    v.fit = generic_fit<In>;
    v.launch = generic_launch<In>;
    v.prepare = no_prepare;
    return v;
}

void register_generic(std::vector<Variant> &r) {
    r.push_back(make_generic<float>(
        "generic_f32: 1x256 DMsxsamples/CTA, 1x1 outputs/thread, global reads, no reuse",
        DEDISP_F32));
    r.push_back(make_generic<uint8_t>(
        "generic_u8: 1x256 DMsxsamples/CTA, 1x1 outputs/thread, global reads, no reuse",
        DEDISP_U8));
}

}  // namespace dedisp

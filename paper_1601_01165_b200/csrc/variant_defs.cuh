// variant_defs.cuh -- turns a kernel instantiation into a registry entry (step a8: the set of
// tunable configurations the auto-tuner sweeps).  The list of instantiations lives in
// ONE place, variants.py; build.py generates one translation unit per entry plus the registry table
// (build/registry_gen.inc) from it.
#pragma once
#include <cstdio>

#include "kernel_tree.cuh"
#include "kernels.cuh"

namespace dedisp {

constexpr size_t kMaxSmem = 227 * 1024;

// ---------------------------------------------------------------- generic (no reuse)
template <typename In>
VariantFit generic_fit(const Variant &v, const PlanShape &p, int) {
    VariantFit f;
    f.ok = p.dtype == v.dtype && p.D <= 65535;
    return f;
}
template <typename In>
cudaError_t generic_launch(const KArgs &a, int nr_beams, size_t, cudaStream_t st) {
    dim3 grid((a.S + 255) / 256, a.D, nr_beams);
    generic_kernel<In><<<grid, 256, 0, st>>>(a);
    return cudaGetLastError();
}
inline cudaError_t no_prepare(size_t) { return cudaSuccess; }

template <typename In>
Variant make_generic() {
    static char name[96];
    const bool u8 = sizeof(In) == 1;
    snprintf(name, sizeof name,
             "generic_%s: 1x256 DMsxsamples/CTA, 1x1 outputs/thread, global reads, no reuse",
             u8 ? "u8" : "f32");
    Variant v;
    v.name = name;
    v.dtype = u8 ? DEDISP_U8 : DEDISP_F32;
    v.kind = KIND_GENERIC;
    v.dms_cta = 1;
    v.samples_cta = 256;
    v.dt = v.tt = 1;
    v.cc = 0;
    v.stages = 0;
    v.qmax = 0;
    v.threads = 256;
    v.fit = generic_fit<In>;
    v.launch = generic_launch<In>;
    v.prepare = no_prepare;
    return v;
}

// ---------------------------------------------------------------- lds (staged tile, 1 word per add)
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

// The attribute belongs to the kernel, not to a plan: it is set to the most any plan may ask for (the
// fit functions refuse more than kMaxSmem), so that preparing the variant for a second, smaller plan does
// not lower the limit under a live plan that needs more.
template <typename T>
cudaError_t tiled_prepare(size_t) {
    return cudaFuncSetAttribute(tiled_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)kMaxSmem);
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
    v.kind = KIND_LDS;
    v.dms_cta = T::DMS_CTA;
    v.samples_cta = T::SAMPLES_CTA;
    v.dt = T::DT;
    v.tt = T::TT;
    v.cc = T::CC;
    v.stages = T::NSTAGE;
    v.qmax = 0;
    v.threads = T::THREADS;
    v.fit = tiled_fit<T>;
    v.launch = tiled_launch<T>;
    v.prepare = tiled_prepare<T>;
    return v;
}

// ---------------------------------------------------------------- tree (register window + lattice)
template <typename T>
VariantFit tree_fit(const Variant &v, const PlanShape &p, int span_cta) {
    VariantFit f;
    if (p.dtype != v.dtype || !p.tree) return f;
    if (!p.tree->valid || p.tree->qmax > T::QMAX) return f;
    if (p.C > 65535) return f;  // grid.y of desc_kernel
    // staged elements per row: the time tile, the tile's shift span, the align-down slack and the
    // window over-read past the last offset a descriptor can hold
    long lrow = (long)T::HALF + span_cta + 2 * T::AL + T::WNMAX;
    lrow = (lrow + T::AL - 1) / T::AL * T::AL;
    if (span_cta + T::AL > 0x3fff) return f;  // window offsets are 14-bit descriptor fields
    size_t smem = tree_smem_bytes<T>((int)lrow);
    if (smem > kMaxSmem) return f;
    const long span_t = T::U8 ? p.S2 : p.S;  // elements along time the grid has to cover
    if ((span_t + T::HALF - 1) / T::HALF > 65535) return f;
    f.ok = true;
    f.lrow = (int)lrow;
    f.smem = smem;
    return f;
}

// Persistent CTAs (kernel_tree.cuh): as many as fit the device at once, each working through every
// (SMs x CTAs per SM)-th tile.
inline int device_sm_count() {
    static int sms[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64) dev = 0;
    if (!sms[dev]) cudaDeviceGetAttribute(&sms[dev], cudaDevAttrMultiProcessorCount, dev);
    return sms[dev] > 0 ? sms[dev] : 1;
}

template <typename T>
cudaError_t tree_launch(const KArgs &a0, int nr_beams, size_t smem, cudaStream_t st) {
    KArgs a = a0;
    const int nt = T::U8 ? a.S2 : a.S;  // pairs / samples along time
    a.nx = (a.D + T::DMS_CTA - 1) / T::DMS_CTA;
    a.ny = (nt + T::HALF - 1) / T::HALF;
    const long long tiles = (long long)a.nx * a.ny * nr_beams;
    if (tiles > 0x7fffffffLL) return cudaErrorInvalidValue;
    a.ntiles = (int)tiles;
    // fp32: persistent CTAs (0.9 % faster: the next tile's first chunks are in flight while a tile's last
    // ones are added and its results stored).  uint8: one CTA per tile on a 3-D grid (persistent CTAs
    // measured 1 % slower there).
    dim3 grid((unsigned)a.nx, (unsigned)a.ny, (unsigned)nr_beams);
    if (T::PERSIST) {
        const long long resident = (long long)device_sm_count() * T::MINB;
        grid = dim3((unsigned)(tiles < resident ? tiles : resident), 1, 1);
    }
    tree_kernel<T><<<grid, T::THREADS, smem, st>>>(a, a.desc, a.descpitch);
    return cudaGetLastError();
}

template <typename T>
cudaError_t tree_prepare(size_t) {   // see tiled_prepare
    return cudaFuncSetAttribute(tree_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)kMaxSmem);
}

template <typename T>
Variant make_tree() {
    static char name[112];
    snprintf(name, sizeof name,
             "tree_%s: %dx%d DMsxsamples/CTA, %dx%d outputs/thread, cc%d s%d q%d b%d%s",
             T::U8 ? "u8" : "f32", T::DMS_CTA, T::SAMPLES_CTA, T::DT, T::U8 ? 2 * T::TT : T::TT, T::CC,
             T::NSTAGE, T::QMAX, T::MINB, T::LAZY ? " lazy" : "");
    Variant v;
    v.name = name;
    v.dtype = T::U8 ? DEDISP_U8 : DEDISP_F32;
    v.kind = KIND_TREE;
    v.dms_cta = T::DMS_CTA;
    v.samples_cta = T::SAMPLES_CTA;
    v.dt = T::DT;
    v.tt = T::U8 ? 2 * T::TT : T::TT;
    v.cc = T::CC;
    v.stages = T::NSTAGE;
    v.qmax = T::QMAX;
    v.lazy = T::LAZY;
    v.threads = T::THREADS;
    v.fit = tree_fit<T>;
    v.launch = tree_launch<T>;
    v.prepare = tree_prepare<T>;
    return v;
}

}  // namespace dedisp

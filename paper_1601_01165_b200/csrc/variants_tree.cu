// variants_tree.cu -- KIND_TREE instantiations (fp32): register window + generated branch lattice.
// TT = 12, 20, 28 keep the LDS.128 window loads bank-conflict free (lane stride is an odd number
// of 16-byte chunks).  The (DT, TT, QMAX) triples must be listed in build.py's TREE_COMBOS.
#include "kernel_tree.cuh"
#include "variants_common.cuh"

namespace dedisp {

template <typename T>
static VariantFit tree_fit(const Variant &v, const PlanShape &p, int span_cta) {
    VariantFit f;
    if (p.dtype != v.dtype || !p.tree) return f;
    if (!p.tree->valid || p.tree->qmax > T::QMAX) return f;
    const TreeTable *t = p.tree->find(T::DT, T::DMS_CTA);
    if (!t || !t->valid) return f;
    // uint8 sums are accumulated in fp32: exact while C * 255 < 2^24
    if (T::U8 && (long)p.C * 255 >= (1L << 24)) return f;
    long lrow = (long)T::SAMPLES_CTA + span_cta + 2 * T::AL + T::WNMAX;
    lrow = (lrow + T::AL - 1) / T::AL * T::AL;
    size_t smem = tree_smem_bytes<T>((int)lrow);
    if (smem > kMaxSmem) return f;
    if ((p.S + T::SAMPLES_CTA - 1) / T::SAMPLES_CTA > 65535) return f;
    f.ok = true;
    f.lrow = (int)lrow;
    f.smem = smem;
    return f;
}

template <typename T>
static cudaError_t tree_launch(const KArgs &a, int nr_beams, size_t smem, cudaStream_t st) {
    dim3 grid((a.D + T::DMS_CTA - 1) / T::DMS_CTA, (a.S + T::SAMPLES_CTA - 1) / T::SAMPLES_CTA,
              nr_beams);
    tree_kernel<T><<<grid, T::THREADS, smem, st>>>(a, a.desc, a.descpitch);
    return cudaGetLastError();
}

template <typename T>
static cudaError_t tree_prepare(size_t smem) {
    return cudaFuncSetAttribute(tree_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)smem);
}

template <typename T>
static Variant make_tree() {
    static char name[112];
    snprintf(name, sizeof name,
             "tree_%s: %dx%d DMsxsamples/CTA, %dx%d outputs/thread, cc%d s%d q%d b%d",
             T::U8 ? "u8" : "f32", T::DMS_CTA, T::SAMPLES_CTA, T::DT, T::TT, T::CC, T::NSTAGE, T::QMAX, T::MINB);
    Variant v;
    v.name = name;
    v.dtype = T::U8 ? DEDISP_U8 : DEDISP_F32;
    v.kind = KIND_TREE;
    v.dms_cta = T::DMS_CTA;
    v.samples_cta = T::SAMPLES_CTA;
    v.dt = T::DT;
    v.tt = T::TT;
    v.cc = T::CC;
    v.stages = T::NSTAGE;
    v.rstep = T::QMAX;
    v.threads = T::THREADS;
    v.fit = tree_fit<T>;
    v.launch = tree_launch<T>;
    v.prepare = tree_prepare<T>;
    return v;
}

// One variant per translation unit (-DTREE_PART=i): build.py reads this list for the parts and for
// the (DT, TT, QMAX) lattices gen_tree.py must emit.
//    part  input   WD WT DT TT CC NS QMAX MINB        DMs x samples per CTA
#define TREE_VARIANTS(X)                                                  \
    X(0, float, 8, 1, 8, 20, 8, 4, 3, 1)    /* 64 x 640  */                \
    X(1, float, 4, 2, 8, 20, 8, 4, 3, 1)    /* 32 x 1280 */                \
    X(2, float, 8, 1, 4, 28, 8, 4, 4, 1)    /* 32 x 896  */                \
    X(3, float, 12, 1, 4, 20, 8, 4, 4, 1)   /* 48 x 640  */                \
    X(4, float, 16, 1, 6, 12, 8, 4, 4, 1)   /* 96 x 384  */                \
    X(5, float, 12, 1, 8, 12, 8, 4, 4, 1)   /* 96 x 384  */                \
    X(6, float, 8, 1, 4, 12, 8, 3, 4, 2)    /* 32 x 384, 2 CTAs/SM */      \
    X(7, float, 8, 1, 6, 20, 8, 4, 4, 1)    /* 48 x 640  */                \
    X(8, float, 8, 1, 8, 20, 8, 4, 4, 1)    /* 64 x 640, q <= 4 */         \
    X(9, float, 8, 1, 6, 28, 8, 4, 3, 1)    /* 48 x 896 */                 \
    X(10, float, 8, 1, 8, 20, 4, 6, 3, 1)   /* 64 x 640, cc4 s6 */         \
    X(11, float, 4, 1, 4, 12, 8, 3, 4, 4)   /* 16 x 384, small problems */ \
    X(12, uint8_t, 8, 1, 8, 20, 8, 4, 4, 1) /* 64 x 640  */                \
    X(13, uint8_t, 16, 1, 6, 12, 8, 4, 4, 1) /* 96 x 384 */                \
    X(14, uint8_t, 8, 1, 6, 28, 8, 4, 4, 1) /* 48 x 896  */                \
    X(15, uint8_t, 4, 1, 4, 12, 8, 3, 4, 4) /* 16 x 384, small problems */ \
    X(16, float, 12, 1, 4, 28, 8, 4, 3, 1)  /* 48 x 896, 12 warps */       \
    X(17, float, 8, 1, 5, 36, 8, 4, 3, 1)   /* 40 x 1152 */                \
    X(18, float, 8, 1, 4, 44, 8, 3, 3, 1)   /* 32 x 1408 */                \
    X(19, float, 12, 1, 5, 20, 8, 4, 3, 1)  /* 60 x 640, 12 warps */       \
    X(20, float, 8, 1, 6, 28, 16, 2, 3, 1)  /* 48 x 896, cc16 s2 */        \
    X(21, float, 8, 1, 6, 28, 4, 6, 3, 1)   /* 48 x 896, cc4 s6 */         \
    X(22, uint8_t, 12, 1, 4, 20, 8, 4, 4, 1) /* 48 x 640, 12 warps */      \
    X(23, uint8_t, 12, 1, 4, 28, 8, 4, 3, 1) /* 48 x 896, 12 warps, q <= 3 */ \
    X(24, uint8_t, 8, 1, 8, 20, 8, 4, 3, 1)  /* 64 x 640, q <= 3 */        \
    X(25, uint8_t, 16, 1, 4, 12, 8, 4, 4, 1) /* 64 x 384, 16 warps */      \
    X(26, float, 12, 1, 4, 28, 16, 3, 3, 1) /* 48 x 896, 12 warps, cc16 s3 */ \
    X(27, float, 8, 1, 6, 28, 16, 3, 3, 1)  /* 48 x 896, cc16 s3 */        \
    X(28, float, 12, 1, 4, 28, 12, 4, 3, 1) /* 48 x 896, 12 warps, cc12 s4 */ \
    X(29, float, 12, 1, 5, 20, 16, 3, 3, 1) /* 60 x 640, 12 warps, cc16 s3 */ \
    X(30, float, 12, 1, 4, 20, 16, 3, 4, 1) /* 48 x 640, 12 warps, cc16 s3, q <= 4 */ \
    X(31, float, 16, 1, 6, 12, 16, 3, 4, 1) /* 96 x 384, 16 warps, cc16 s3, q <= 4 */

#ifndef TREE_PART
#define TREE_PART 0
#endif
#define DEDISP_CAT(a, b) a##b
#define DEDISP_TREE_REG(P) DEDISP_CAT(register_tree, P)
template <int P> struct TreePart;
#define X(P, IN, WD, WT, DT, TT, CC, NS, QMAX, MINB) \
    template <> struct TreePart<P> { typedef TreeTile<IN, WD, WT, DT, TT, CC, NS, QMAX, MINB> type; };
TREE_VARIANTS(X)
#undef X
void DEDISP_TREE_REG(TREE_PART)(std::vector<Variant> &r) {
    r.push_back(make_tree<TreePart<TREE_PART>::type>());
}
}  // namespace dedisp

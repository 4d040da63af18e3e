// kernel_tree.cuh -- KIND_TREE: the register-window kernel whose per-DM window offset is selected
// by a generated lattice of warp-uniform two-way branches (gen_tree.py) instead of a switch.
//
// Steps a4-a6 of SURVEY.md 8(a), Algorithm 1.  The reuse the paper gets from
// local memory is taken one level further down: every shared-memory word a thread
// loads feeds about DT adds from registers, because shared memory delivers 32 words/clk/SM while
// the fp32 pipes retire 128 adds/clk/SM.
//
//   CTA tile   : DMS_CTA = WD*DT DMs  x  SAMPLES_CTA = WT*32*TT samples; NW = WD*WT warps, no
//                dedicated producer warp (its registers would be wasted at ~240 registers/thread):
//                warp (k mod NW) issues the bulk copies of chunk k + NSTAGE - 1 when it has
//                finished chunk k.
//   per thread : DT adjacent DMs x TT consecutive samples in registers.
//   per channel: one descriptor word per (channel, DM group) built at plan creation
//                (desc_kernel, shift_table.cu):  [31:16] window offset in the staged row
//                [15:8] 1 << q_c   [7:0] bits, the group's shift increments being q_c + bit_j.
//                Staged per chunk next to the input rows.
#pragma once
#include "kernels.cuh"
#include "build/tree_gen.cuh"

namespace dedisp {

template <typename In_, int WD_, int WT_, int DT_, int TT_, int CC_, int NSTAGE_, int QMAX_,
          int MINB_>
struct TreeTile {
    typedef In_ In;                              // float, or uint8_t converted to fp32 at staging
    typedef typename AccOf<In_>::type Acc;       // output type: float / uint32_t
    static constexpr bool U8 = sizeof(In_) == 1;
    static constexpr int AL = 16 / (int)sizeof(In_);  // elements per 16 bytes of input
    static constexpr int WD = WD_, WT = WT_, DT = DT_, TT = TT_, CC = CC_, NSTAGE = NSTAGE_,
                         QMAX = QMAX_, MINB = MINB_;
    static constexpr int NW = WD * WT;
    static constexpr int THREADS = NW * 32;
    static constexpr int DMS_CTA = WD * DT;
    static constexpr int SAMPLES_CTA = WT * 32 * TT;
    static constexpr int WNMAX = TreeStep<DT, TT, QMAX>::WNMAX;
    static_assert(TT % 4 == 0, "thread windows are loaded with LDS.128");
    static_assert(WD % 4 == 0, "descriptor rows are copied in 16-byte units");
    static_assert(CC <= 32, "one lane per channel of a chunk issues its copies");
    static_assert(DT <= 9 && QMAX <= 7, "8 increment bits and a one-hot q per descriptor");
    static_assert(SAMPLES_CTA % AL == 0, "time tiles start on 16-byte boundaries of the input");
};

// Shared memory (dynamic): mbarriers | NSTAGE stages { CC input rows of lrow elements | CC x WD
// descriptors } | for uint8 input three fp32 buffers { CC rows of lrow floats | CC x WD descriptors }
// the compute loop reads (the stage rows are converted into them, chunk k into buffer k % 3, one
// chunk ahead of the adds).
template <typename T>
__host__ __device__ inline size_t tree_stage_bytes(int lrow) {
    return (size_t)T::CC * ((size_t)lrow * sizeof(typename T::In) + (size_t)T::WD * 4);
}
template <typename T>
__host__ __device__ inline size_t tree_fbuf_bytes(int lrow) {
    return (size_t)T::CC * ((size_t)lrow * 4 + (size_t)T::WD * 4);
}
template <typename T>
__host__ __device__ inline size_t tree_smem_bytes(int lrow) {
    return T::NSTAGE * tree_stage_bytes<T>(lrow) + (T::U8 ? 3 * tree_fbuf_bytes<T>(lrow) : 0) +
           (2 * T::NSTAGE + 3) * sizeof(uint64_t) + 16 + T::WD * 4;
}

// Issue the copies of chunk k into its stage (called by one whole warp; lane l < CC stages channel
// k*CC + l: its input span and its WD descriptors).
template <typename T>
__device__ __forceinline__ void tree_issue(const KArgs &a, const typename T::In *in,
                                           const uint32_t *desc,
                                           int descpitch, int k, int lane, int T0, int dm_lo,
                                           int g_lo, unsigned char *stages, size_t sbytes,
                                           size_t data_bytes, uint64_t *full) {
    const int s = k % T::NSTAGE;
    const int c = k * T::CC + lane;
    uint32_t bytes = 0;
    if (lane < T::CC && c < a.C) {
        const int32_t *trow = a.shiftT + (size_t)c * a.dpitch + dm_lo;
        const int smin = trow[0], smax = trow[T::DMS_CTA - 1];
        const int g0 = T0 + (smin & ~(T::AL - 1));
        int end = T0 + T::SAMPLES_CTA + smax;
        end = end < a.in_pitch ? end : a.in_pitch;
        int len = (end - g0 + T::AL - 1) & ~(T::AL - 1);
        len = len < a.lrow ? len : a.lrow;
        unsigned char *st = stages + (size_t)s * sbytes;
        const uint32_t nb = (uint32_t)len * sizeof(typename T::In);
        bulk_g2s(st + (size_t)lane * a.lrow * sizeof(typename T::In),
                 in + (size_t)c * a.in_pitch + g0, nb, &full[s]);
        bulk_g2s(st + data_bytes + (size_t)lane * T::WD * 4, desc + (size_t)c * descpitch + g_lo,
                 T::WD * 4, &full[s]);
        bytes = nb + T::WD * 4;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) bytes += __shfl_xor_sync(0xffffffffu, bytes, o);
    if (lane == 0) mbar_arrive_expect_tx(&full[s], bytes);
}

// grid: x = DM tiles (fastest: CTAs resident together share input time ranges in L2), y = time
// tiles, z = beams.
template <typename T>
__global__ void __launch_bounds__(T::THREADS, T::MINB) tree_kernel(KArgs a, const uint32_t *desc,
                                                             int descpitch) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw);
    uint64_t *empty = full + T::NSTAGE;
    uint64_t *conv = empty + T::NSTAGE;  // uint8 input: fp32 buffer b holds a converted chunk
    unsigned char *stages =
        smem_raw + (((2 * T::NSTAGE + 3) * sizeof(uint64_t) + 15) & ~(size_t)15);
    const size_t sbytes = tree_stage_bytes<T>(a.lrow);
    const size_t data_bytes = (size_t)T::CC * a.lrow * sizeof(typename T::In);

    // Everything derived from the warp index -- the warp's DM group, its descriptors, every lattice
    // test -- is warp-uniform: the lattice branches never diverge.
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int dm_lo = blockIdx.x * T::DMS_CTA;
    const int g_lo = blockIdx.x * T::WD;
    const int T0 = blockIdx.y * T::SAMPLES_CTA;
    const int nchunks = (a.C + T::CC - 1) / T::CC;
    const typename T::In *in =
        (const typename T::In *)a.in + (size_t)blockIdx.z * a.C * a.in_pitch;

    if (threadIdx.x == 0) {
        for (int s = 0; s < T::NSTAGE; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], T::NW);
        }
        for (int b = 0; b < 3; ++b) mbar_init(&conv[b], T::NW);
        mbar_fence_init();
    }
    __syncthreads();
    // prologue: warp 0 fills the first NSTAGE-1 stages (all NSTAGE for uint8 input, whose stages
    // are released one chunk early, after conversion)
    constexpr int AHEAD = T::U8 ? T::NSTAGE : T::NSTAGE - 1;
    if (warp == 0)
        for (int k = 0; k < AHEAD && k < nchunks; ++k)
            tree_issue<T>(a, in, desc, descpitch, k, lane, T0, dm_lo, g_lo, stages, sbytes,
                          data_bytes, full);

    const int g = warp % T::WD;                  // DM group
    const int tw = (warp / T::WD) * 32 * T::TT;  // first sample of the warp's time chunk
    float acc[T::DT][T::TT];
#pragma unroll
    for (int j = 0; j < T::DT; ++j)
#pragma unroll
        for (int k = 0; k < T::TT; ++k) acc[j][k] = 0.f;

    // uint8 input: convert chunk k's rows to fp32 (exact; sums stay below 2^24, checked at plan
    // creation) into buffer k % 3, copy its descriptors, release the stage.  Every warp converts a
    // slice; conv[k % 3] completes when all have.
    auto convert = [&](int k) {
        const int s = k % T::NSTAGE;
        mbar_wait(&full[s], (k / T::NSTAGE) & 1);
        const unsigned char *st = stages + (size_t)s * sbytes;
        const int ncc = (a.C - k * T::CC) < T::CC ? (a.C - k * T::CC) : T::CC;
        unsigned char *fb = stages + T::NSTAGE * sbytes + (size_t)(k % 3) * tree_fbuf_bytes<T>(a.lrow);
        float4 *frow = reinterpret_cast<float4 *>(fb);
        const uint4 *raw = reinterpret_cast<const uint4 *>(st);
        const int n16 = ncc * a.lrow / 16;  // 16 samples per 128-bit load (lrow is a multiple of 16)
        for (int i = threadIdx.x; i < n16; i += T::THREADS) {
            const uint4 x = raw[i];
            const uint32_t xs[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                // byte b -> float: 0x4B000000 | b is 2^23 + b; subtract 2^23 (two at a time)
                float4 v;
                v.x = __uint_as_float(__byte_perm(xs[m], 0x4B000000u, 0x7650));
                v.y = __uint_as_float(__byte_perm(xs[m], 0x4B000000u, 0x7651));
                v.z = __uint_as_float(__byte_perm(xs[m], 0x4B000000u, 0x7652));
                v.w = __uint_as_float(__byte_perm(xs[m], 0x4B000000u, 0x7653));
                asm("{.reg .b64 a, b; mov.b64 a, {%0, %1}; mov.b64 b, {%2, %2}; add.f32x2 a, a, b; "
                    "mov.b64 {%0, %1}, a;}" : "+f"(v.x), "+f"(v.y) : "f"(-8388608.f));
                asm("{.reg .b64 a, b; mov.b64 a, {%0, %1}; mov.b64 b, {%2, %2}; add.f32x2 a, a, b; "
                    "mov.b64 {%0, %1}, a;}" : "+f"(v.z), "+f"(v.w) : "f"(-8388608.f));
                frow[4 * i + m] = v;
            }
        }
        uint32_t *fds = reinterpret_cast<uint32_t *>(fb + (size_t)T::CC * a.lrow * 4);
        if ((int)threadIdx.x < ncc * T::WD)
            fds[threadIdx.x] = reinterpret_cast<const uint32_t *>(st + data_bytes)[threadIdx.x];
        __syncwarp();
        if (lane == 0) {
            mbar_arrive(&conv[k % 3]);
            mbar_arrive(&empty[s]);
        }
    };
    if constexpr (T::U8) convert(0);

    for (int k = 0; k < nchunks; ++k) {
        const int s = k % T::NSTAGE;
        const int ncc = (a.C - k * T::CC) < T::CC ? (a.C - k * T::CC) : T::CC;
        const float *rows;
        const uint32_t *ds;
        if constexpr (T::U8) {
            // all warps have converted chunk k, so all have finished the adds of chunk k-2, whose
            // buffer chunk k+1 is converted into now
            mbar_wait(&conv[k % 3], (k / 3) & 1);
            if (k + 1 < nchunks) convert(k + 1);
            const unsigned char *fb =
                stages + T::NSTAGE * sbytes + (size_t)(k % 3) * tree_fbuf_bytes<T>(a.lrow);
            rows = reinterpret_cast<const float *>(fb) + tw + lane * T::TT;
            ds = reinterpret_cast<const uint32_t *>(fb + (size_t)T::CC * a.lrow * 4) + g;
        } else {
            mbar_wait(&full[s], (k / T::NSTAGE) & 1);
            const unsigned char *st = stages + (size_t)s * sbytes;
            rows = reinterpret_cast<const float *>(st) + tw + lane * T::TT;
            ds = reinterpret_cast<const uint32_t *>(st + data_bytes) + g;
        }
        TreeStep<T::DT, T::TT, T::QMAX>::template chunk<T::WD>(acc, rows, ds, ncc, a.lrow);
        if constexpr (!T::U8) {
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[s]);
        }
        // producer duty, rotating over the warps (step a4): refill the most recently released
        // stage, which the other warps have normally left by now
        const int kk = k + AHEAD;
        if (kk < nchunks && warp == k % T::NW) {
            if (kk >= T::NSTAGE) mbar_wait(&empty[kk % T::NSTAGE], ((kk / T::NSTAGE) - 1) & 1);
            tree_issue<T>(a, in, desc, descpitch, kk, lane, T0, dm_lo, g_lo, stages, sbytes,
                          data_bytes, full);
        }
    }

    // store (step a6): each thread writes TT consecutive samples of each of its DMs
    typedef typename T::Acc Acc;
    Acc *out = (Acc *)a.out + (size_t)blockIdx.z * a.D * a.S;
    const int dm0 = dm_lo + g * T::DT;
    const int t0 = T0 + tw + lane * T::TT;
    const bool vec = (a.S & 3) == 0 && t0 + T::TT <= a.S;
#pragma unroll
    for (int j = 0; j < T::DT; ++j) {
        if (dm0 + j >= a.D) break;
        Acc *o = out + (size_t)(dm0 + j) * a.S + t0;
        if (vec) {
#pragma unroll
            for (int k = 0; k < T::TT; k += 4) {
                if constexpr (T::U8)
                    *reinterpret_cast<uint4 *>(o + k) =
                        make_uint4(__float2uint_rn(acc[j][k]), __float2uint_rn(acc[j][k + 1]),
                                   __float2uint_rn(acc[j][k + 2]), __float2uint_rn(acc[j][k + 3]));
                else
                    *reinterpret_cast<float4 *>(o + k) =
                        make_float4(acc[j][k], acc[j][k + 1], acc[j][k + 2], acc[j][k + 3]);
            }
        } else {
#pragma unroll
            for (int k = 0; k < T::TT; ++k)
                if (t0 + k < a.S) {
                    if constexpr (T::U8) o[k] = __float2uint_rn(acc[j][k]);
                    else o[k] = acc[j][k];
                }
        }
    }
}

}  // namespace dedisp

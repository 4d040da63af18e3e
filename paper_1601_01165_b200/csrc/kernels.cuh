// kernels.cuh -- steps a4-a7: the dedispersion kernels, Algorithm 1
// (PAPER.md:51-55): out[b][i][t] = sum_c in[b][c][t + shift(c, dm_i)].
//
//   generic_kernel : one (DM, sample) per thread, global reads (the paper's "generically tuned"
//                    baseline).
//   tiled_kernel   : each CTA owns DMs_CTA x SAMPLES_CTA outputs.  A producer warp stages, per
//                    channel of a chunk, the contiguous input span covering the DM tile's shift range
//                    into shared memory with 1-D bulk async copies (cp.async.bulk, SASS UBLKCP)
//                    completing on an mbarrier ring; consumer warps accumulate DT x TT outputs
//                    per thread in registers (work-items computing several
//                    elements, data reuse through local memory), one shared-memory word per add,
//                    lanes on consecutive samples (KIND_LDS).
// The register-window kernels (KIND_TREE) are in kernel_tree.cuh.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "dedisp_internal.h"

namespace dedisp {

// ---------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    uint32_t addr = smem_u32(bar);
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(addr),
        "r"(parity)
        : "memory");
}
// 1-D bulk async copy global -> shared, completion counted in bytes on an mbarrier.
// dst, src and bytes are multiples of 16.
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes,
                                         uint64_t *bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
            "r"(smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

template <typename In> struct AccOf;
template <> struct AccOf<float> { typedef float type; };
template <> struct AccOf<uint8_t> { typedef uint32_t type; };

// ---------------------------------------------------------------- generic (no reuse)
// grid: x = ceil(S / 256), y = D, z = beams; 256 threads, one output each.  All lanes of a warp
// share the DM, so the table read is a broadcast and the input read is coalesced but unaligned
// (PAPER.md:72).
template <typename In>
__global__ void __launch_bounds__(256) generic_kernel(KArgs a) {
    typedef typename AccOf<In>::type Acc;
    int t = blockIdx.x * 256 + threadIdx.x;
    int i = blockIdx.y;
    if (t >= a.S) return;
    const In *in = (const In *)a.in + (size_t)blockIdx.z * a.C * a.in_pitch;
    const int32_t *sh = a.shift + (size_t)i * a.C;
    Acc acc = 0;
    for (int c = 0; c < a.C; ++c) acc += (Acc)in[(size_t)c * a.in_pitch + t + sh[c]];
    ((Acc *)a.out)[((size_t)blockIdx.z * a.D + i) * a.S + t] = acc;
}

// ---------------------------------------------------------------- tiled kernels
// Compile-time tile description.
//   WD x WT consumer warps: WD DM groups of DT DMs, WT time chunks of 32*TT samples.
//   CC channels per pipeline stage, NSTAGE stages.
template <typename In_, int WD_, int WT_, int DT_, int TT_, int CC_, int NSTAGE_, int MINB_>
struct Tile {
    typedef In_ In;
    typedef typename AccOf<In_>::type Acc;
    static constexpr int WD = WD_, WT = WT_, DT = DT_, TT = TT_, CC = CC_, NSTAGE = NSTAGE_,
                         MINB = MINB_;
    static constexpr int NW = WD * WT;              // consumer warps
    static constexpr int THREADS = (NW + 1) * 32;   // + producer warp
    static constexpr int DMS_CTA = WD * DT;
    static constexpr int SAMPLES_CTA = WT * 32 * TT;
    static constexpr int AL = 16 / (int)sizeof(In);  // elements per 16 bytes
    static_assert(DMS_CTA % 4 == 0, "shift rows are copied in 16-byte units");
    static_assert(CC <= 32, "one producer lane per channel of a chunk");
};

// Shared-memory carve-up (dynamic): NSTAGE x { CC rows of lrow elements | CC x DMS_CTA shifts },
// then the full/empty mbarriers.
template <typename T>
__host__ __device__ inline size_t stage_bytes(int lrow) {
    return (size_t)T::CC * ((size_t)lrow * sizeof(typename T::In) + (size_t)T::DMS_CTA * 4);
}
template <typename T>
__host__ __device__ inline size_t tile_smem_bytes(int lrow) {
    return T::NSTAGE * stage_bytes<T>(lrow) + 2 * T::NSTAGE * sizeof(uint64_t) + 16;
}

// ---- per-channel inner loops -------------------------------------------------------------
// row : the channel's staged span; element 0 is input sample T0 + (smin & ~(AL-1)) where smin is
//       the shift of the CTA's first DM.  sh : the channel's DMS_CTA shifts (shared memory).
template <typename T>
__device__ __forceinline__ void channel_lds(typename T::Acc (&acc)[T::DT][T::TT],
                                            const typename T::In *row, const int32_t *sh, int g,
                                            int tw, int lane) {
    const int base = sh[0] & ~(T::AL - 1);
    // the group's DT shifts: warp-uniform (broadcast) loads, four at a time where DT allows -- each is
    // a shared-memory wavefront, and wavefronts are what bounds this kernel
    int s[T::DT];
    if constexpr (T::DT % 4 == 0) {
#pragma unroll
        for (int j = 0; j < T::DT; j += 4) {
            const int4 v = *reinterpret_cast<const int4 *>(sh + g * T::DT + j);
            s[j] = v.x; s[j + 1] = v.y; s[j + 2] = v.z; s[j + 3] = v.w;
        }
    } else if constexpr (T::DT % 2 == 0) {
#pragma unroll
        for (int j = 0; j < T::DT; j += 2) {
            const int2 v = *reinterpret_cast<const int2 *>(sh + g * T::DT + j);
            s[j] = v.x; s[j + 1] = v.y;
        }
    } else {
#pragma unroll
        for (int j = 0; j < T::DT; ++j) s[j] = sh[g * T::DT + j];
    }
#pragma unroll
    for (int j = 0; j < T::DT; ++j) {
        const typename T::In *p = row + (s[j] - base) + tw + lane;
#pragma unroll
        for (int k = 0; k < T::TT; ++k) acc[j][k] += (typename T::Acc)p[32 * k];
    }
}

// ---- the tiled kernel --------------------------------------------------------------------
// grid: x = DM tiles (fastest, so CTAs resident together share the same input time range in L2),
//       y = time tiles, z = beams.  block: NW consumer warps + 1 producer warp.
template <typename T>
__global__ void __launch_bounds__(T::THREADS, T::MINB) tiled_kernel(KArgs a) {
    typedef typename T::In In;
    typedef typename T::Acc Acc;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw);
    uint64_t *empty = full + T::NSTAGE;
    unsigned char *stages = smem_raw + ((2 * T::NSTAGE * sizeof(uint64_t) + 15) & ~(size_t)15);
    const size_t sbytes = stage_bytes<T>(a.lrow);
    const size_t data_bytes = (size_t)T::CC * a.lrow * sizeof(In);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int dm_lo = blockIdx.x * T::DMS_CTA;
    const int T0 = blockIdx.y * T::SAMPLES_CTA;
    const int nchunks = (a.C + T::CC - 1) / T::CC;

    if (threadIdx.x == 0) {
        for (int s = 0; s < T::NSTAGE; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], T::NW);
        }
        mbar_fence_init();
    }
    __syncthreads();

    if (warp == T::NW) {
        // ---------------- producer warp: lane l stages channel l of each chunk (step a4)
        const In *in = (const In *)a.in + (size_t)blockIdx.z * a.C * a.in_pitch;
        for (int k = 0; k < nchunks; ++k) {
            const int s = k % T::NSTAGE, use = k / T::NSTAGE;
            if (use > 0) mbar_wait(&empty[s], (use - 1) & 1);
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
                const uint32_t nb = (uint32_t)len * sizeof(In);
                bulk_g2s(st + (size_t)lane * a.lrow * sizeof(In),
                         in + (size_t)c * a.in_pitch + g0, nb, &full[s]);
                bulk_g2s(st + data_bytes + (size_t)lane * T::DMS_CTA * 4, trow, T::DMS_CTA * 4,
                         &full[s]);
                bytes = nb + T::DMS_CTA * 4;
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) bytes += __shfl_xor_sync(0xffffffffu, bytes, o);
            if (lane == 0) mbar_arrive_expect_tx(&full[s], bytes);
        }
        return;
    }

    // ---------------- consumer warps (steps a5, a6)
    const int g = warp % T::WD;              // DM group
    const int tw = (warp / T::WD) * 32 * T::TT;  // first sample of the warp's time chunk
    Acc acc[T::DT][T::TT];
#pragma unroll
    for (int j = 0; j < T::DT; ++j)
#pragma unroll
        for (int k = 0; k < T::TT; ++k) acc[j][k] = 0;

    for (int k = 0; k < nchunks; ++k) {
        const int s = k % T::NSTAGE, use = k / T::NSTAGE;
        mbar_wait(&full[s], use & 1);
        const unsigned char *st = stages + (size_t)s * sbytes;
        const In *rows = reinterpret_cast<const In *>(st);
        const int32_t *shs = reinterpret_cast<const int32_t *>(st + data_bytes);
        const int ncc = (a.C - k * T::CC) < T::CC ? (a.C - k * T::CC) : T::CC;
        if (ncc == T::CC) {
#pragma unroll 1
            for (int cc = 0; cc < T::CC; ++cc) {
                channel_lds<T>(acc, rows + (size_t)cc * a.lrow, shs + cc * T::DMS_CTA, g, tw, lane);
            }
        } else {
#pragma unroll 1
            for (int cc = 0; cc < ncc; ++cc) {
                channel_lds<T>(acc, rows + (size_t)cc * a.lrow, shs + cc * T::DMS_CTA, g, tw, lane);
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);
    }

    // ---------------- store (step a6): aligned, contiguous per thread / per warp
    Acc *out = (Acc *)a.out + (size_t)blockIdx.z * a.D * a.S;
    const int dm0 = dm_lo + g * T::DT;
    const int t0 = T0 + tw + lane;
#pragma unroll
    for (int j = 0; j < T::DT; ++j) {
        if (dm0 + j >= a.D) break;
        Acc *o = out + (size_t)(dm0 + j) * a.S + t0;
#pragma unroll
        for (int k = 0; k < T::TT; ++k)
            if (t0 + 32 * k < a.S) o[32 * k] = acc[j][k];
    }
}

}  // namespace dedisp

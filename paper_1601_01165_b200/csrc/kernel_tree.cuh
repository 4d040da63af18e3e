// kernel_tree.cuh -- the register-window kernels whose per-DM window offset is selected by a
// generated lattice of warp-uniform two-way branches (gen_tree.py) instead of a switch.
//
// Steps a4-a6 of SURVEY.md 8(a), Algorithm 1.  The reuse the paper gets from
// local memory is taken one level further down: every shared-memory word a thread
// loads feeds about DT adds from registers, because shared memory delivers 32 words/clk/SM while
// the fp32 pipes retire 128 adds/clk/SM.
//
//   CTA tile   : DMS_CTA = WD*DT DMs  x  SAMPLES_CTA samples; NW = WD*WT warps, no dedicated
//                producer warp (its registers would be wasted at ~170-240 registers/thread):
//                warp (k mod NW) issues the bulk copies of a later chunk when it has finished
//                chunk k.
//   per thread : DT adjacent DMs x TT consecutive ELEMENTS in registers.
//                fp32 input : element = one sample; a CTA covers SAMPLES_CTA = HALF = WT*32*TT samples.
//                uint8 input: element = a PAIR of samples S2 = ~S/2 apart, kept as two 16-bit counters
//                in one 32-bit word.  pack_pairs_kernel (shift_table.cu) first rewrites the input as
//                pairs[c][y] = in[c][y] | in[c][y + S2] << 16 in a plan-owned workspace, so one 32-bit
//                integer add accumulates two outputs (t and t + S2) whatever the shift, odd or even;
//                a CTA covers outputs [T0, T0 + HALF) and [S2 + T0, S2 + T0 + HALF).  The counters
//                are flushed into the uint32 output every <= 256 channels (256 * 255 < 2^16).
//   per channel: one descriptor word per (channel, DM group), built when the variant is selected
//                (desc_kernel, shift_table.cu; layout in gen_tree.py): the window's byte offset in
//                the staged row, the first DM's offset in its 16-byte quad, the channel's slope
//                class q_c one-hot, and the bits b_j, the group's shift increments being q_c + b_j.
//                Staged per chunk next to the rows; the row after the chunk's last channel is zero
//                and ends the channel loop.
#pragma once
#include <type_traits>

#include "kernels.cuh"
#ifdef DEDISP_TREE_GEN
#include DEDISP_TREE_GEN          // the one lattice this translation unit instantiates (build.py)
#else
#include "build/tree_gen_common.cuh"
#endif

namespace dedisp {

template <typename In_, int WD_, int WT_, int DT_, int TT_, int CC_, int NSTAGE_, int QMAX_,
          int MINB_, int LAZY_ = 0>
struct TreeTile {
    typedef In_ In;                              // float or uint8_t
    typedef typename AccOf<In_>::type Acc;       // output type: float / uint32_t
    static constexpr bool U8 = sizeof(In_) == 1;
    // what a window register / accumulator register holds: a float, or a pair of 16-bit counters
    typedef typename std::conditional<U8, uint32_t, float>::type Elem;
    typedef Elem Stg;                            // what a staged row holds (4 bytes either way)
    static constexpr int AL = 4;                 // staged elements per 16 bytes
    static constexpr int WD = WD_, WT = WT_, DT = DT_, TT = TT_, CC = CC_, NSTAGE = NSTAGE_,
                         QMAX = QMAX_, MINB = MINB_;
    // LAZY = 1: the upper window quads are loaded only on the lattice paths that read them (gen_tree.py)
    static constexpr int LAZY = LAZY_;
    // persistent CTAs (fp32): the chunk ring runs on across the CTA's tiles, see tree_tile
    static constexpr bool PERSIST = !U8;
    static constexpr int NW = WD * WT;
    static constexpr int THREADS = NW * 32;
    static constexpr int DMS_CTA = WD * DT;
    static constexpr int HALF = WT * 32 * TT;    // elements per CTA along time
    static constexpr int SAMPLES_CTA = U8 ? 2 * HALF : HALF;  // outputs per DM and CTA
    static constexpr int FLUSH_CHUNKS = 256 / CC;  // uint8: chunks between counter flushes
    static constexpr int WNMAX = TreeStep<Elem, DT, TT, QMAX, LAZY>::WNMAX;
    static_assert(TT % 4 == 0, "thread windows are loaded with LDS.128");
    static_assert(WD % 4 == 0, "descriptor rows are copied in 16-byte units");
    static_assert(CC <= 32, "one lane per channel of a chunk issues its copies");
    static_assert(DT <= 9 && QMAX <= 7, "8 increment bits and a one-hot q per descriptor");
    static_assert(HALF % AL == 0, "time tiles start on 16-byte boundaries of the staged rows");
    // uint8: what the 16-bit pair counters and the carry-chain adds of gen_tree.py rely on.  A counter takes
    // at most 255 per channel and is flushed every FLUSH_CHUNKS chunks, so it cannot carry into its
    // neighbour; the chains join accumulators k and k + 1, so TT must be even for a chain never to join a
    // valid element with one past the row's end (plan.cu checks the matching run-time conditions:
    // S2 a multiple of 4 and pair_pitch >= S2 + M).
    static_assert(!U8 || FLUSH_CHUNKS * CC * 255 < 65536, "a 16-bit pair counter would overflow between flushes");
    static_assert(!U8 || FLUSH_CHUNKS >= 1, "at least one chunk between flushes");
    static_assert(TT % 2 == 0, "carry chains join accumulators k and k + 1");
};

// Shared memory (dynamic): mbarriers | NSTAGE stages { CC rows of lrow staged elements | (CC + 1) x WD
// descriptors, the last row a terminator }.
template <typename T>
__host__ __device__ inline size_t tree_stage_bytes(int lrow) {
    return (size_t)T::CC * ((size_t)lrow * 4 + (size_t)T::WD * 4) + (size_t)T::WD * 4;
}
template <typename T>
__host__ __device__ inline size_t tree_smem_bytes(int lrow) {
    return T::NSTAGE * tree_stage_bytes<T>(lrow) + 2 * T::NSTAGE * sizeof(uint64_t) + 16 + T::WD * 4;
}

// Special registers read through opaque moves: what is derived from them is recomputed where it is
// used (once per chunk, or in the epilogue) instead of being kept in registers across the channel loop,
// where 80-112 accumulators and a 28-52 register window leave nothing to spare.
__device__ __forceinline__ uint32_t sreg_tid() { uint32_t v; asm volatile("mov.u32 %0, %%tid.x;" : "=r"(v)); return v; }
__device__ __forceinline__ uint32_t sreg_ctaid_x() { uint32_t v; asm volatile("mov.u32 %0, %%ctaid.x;" : "=r"(v)); return v; }
__device__ __forceinline__ uint32_t sreg_nctaid_x() { uint32_t v; asm volatile("mov.u32 %0, %%nctaid.x;" : "=r"(v)); return v; }
__device__ __forceinline__ uint32_t sreg_ctaid_y() { uint32_t v; asm volatile("mov.u32 %0, %%ctaid.y;" : "=r"(v)); return v; }
__device__ __forceinline__ uint32_t sreg_ctaid_z() { uint32_t v; asm volatile("mov.u32 %0, %%ctaid.z;" : "=r"(v)); return v; }
extern __shared__ __align__(128) unsigned char dedisp_smem[];
__device__ __forceinline__ uint32_t smem_base() {   // shared-window address of the dynamic allocation
    return (uint32_t)__cvta_generic_to_shared(dedisp_smem);   // a constant to ptxas: costs no register
}

// mbarriers by shared-window address (the ring's barriers sit at the start of the allocation)
__device__ __forceinline__ void mbar_arrive_s(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait_s(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}

// Layout of the dynamic shared memory, as shared-window byte offsets from its start.
template <typename T> struct TreeSmem {
    static constexpr uint32_t FULL = 0, EMPTY = T::NSTAGE * 8;
    static constexpr uint32_t STAGES = (2 * T::NSTAGE * 8 + 15) & ~15u;
};

// The kernel is PERSISTENT: a CTA works through the tiles blockIdx.x, blockIdx.x + gridDim.x, ... (tile id =
// (beam * ny + time tile) * nx + DM tile, DM tiles fastest: the CTAs running together share input time ranges
// in L2), and its chunk ring runs on across tile boundaries, so the first chunks of the next tile are in
// flight while the last ones of this tile are added and its results stored.  Tile `it` of this CTA:
// uint8 kernels are not persistent (measured 1 % slower): there the grid is (DM tiles, time tiles, beams)
// and a CTA has the one tile its block index names.
template <bool PERSIST>
__device__ __forceinline__ void tree_tile(const KArgs &a, int it, int &tx, int &ty, int &bz) {
    if constexpr (PERSIST) {
        const uint32_t tile = sreg_ctaid_x() + (uint32_t)it * sreg_nctaid_x();
        tx = (int)(tile % (uint32_t)a.nx);
        const uint32_t r = tile / (uint32_t)a.nx;
        ty = (int)(r % (uint32_t)a.ny);
        bz = (int)(r / (uint32_t)a.ny);
    } else {
        tx = (int)sreg_ctaid_x();
        ty = (int)sreg_ctaid_y();
        bz = (int)sreg_ctaid_z();
    }
}
template <bool PERSIST>
__device__ __forceinline__ int tree_my_tiles(const KArgs &a) {   // tiles this CTA works through (>= 1)
    if constexpr (PERSIST)
        return (int)(((uint32_t)a.ntiles - sreg_ctaid_x() + sreg_nctaid_x() - 1) / sreg_nctaid_x());
    else
        return 1;
}

// Issue the copies of ring position g (chunk g % nchunks of the CTA's tile g / nchunks) into its stage
// (called by one whole warp; lane l < CC stages channel k*CC + l: its row span and its WD descriptors).
// The beam's staged-element matrix [C][pitch] is the fp32 input itself, or the uint8 plan's pair workspace.
// Everything is recomputed from the kernel arguments and the block index (see sreg_*): nothing of it lives
// across the channel loop.
template <typename T>
__device__ __forceinline__ void tree_issue(const KArgs &a, const uint32_t *desc, int descpitch, int g, int nchunks) {
    const int lane = sreg_tid() & 31;
    const int it = g / nchunks;
    const int k = g - it * nchunks;   // chunk of tile `it`; the ring position is g
    int tx, ty, bz;
    tree_tile<T::PERSIST>(a, it, tx, ty, bz);
    const int dm_lo = tx * T::DMS_CTA, g_lo = tx * T::WD;
    const int T0 = ty * T::HALF;
    const int pitch = T::U8 ? a.pair_pitch : a.in_pitch;
    const typename T::Stg *rows =
        (const typename T::Stg *)(T::U8 ? (const void *)a.pairs : a.in) + (size_t)bz * a.C * pitch;
    const uint32_t sbytes = (uint32_t)tree_stage_bytes<T>(a.lrow);
    const uint32_t data_bytes = (uint32_t)T::CC * a.lrow * 4;
    const uint32_t base = smem_base();
    const uint32_t st = base + TreeSmem<T>::STAGES + (uint32_t)(g % T::NSTAGE) * sbytes;
    const uint32_t full = base + TreeSmem<T>::FULL + (uint32_t)(g % T::NSTAGE) * 8;
    const int c = k * T::CC + lane;
    uint32_t bytes = 0;
    // ragged last chunk: the descriptor row after its last channel ends the channel loop
    const int ncc = a.C - k * T::CC;
    // (a generic-proxy store into a stage the bulk copies of a later chunk overwrite again: the proxy fence
    // orders it before them)
    if (ncc < T::CC && lane < T::WD) {
        asm volatile("st.shared.u32 [%0], %1;" ::"r"(st + data_bytes + (uint32_t)(ncc * T::WD + lane) * 4), "r"(0u)
                     : "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    if (lane < T::CC && c < a.C) {
        const int32_t *trow = a.shiftT + (size_t)c * a.dpitch + dm_lo;
        const int smin = trow[0], smax = trow[T::DMS_CTA - 1];
        const int g0 = T0 + (smin & ~(T::AL - 1));
        int end = T0 + T::HALF + smax;
        end = end < pitch ? end : pitch;
        int len = (end - g0 + T::AL - 1) & ~(T::AL - 1);
        len = len < a.lrow ? len : a.lrow;
        len = len > 0 ? len : 0;
        const uint32_t nb = (uint32_t)len * 4;
        if (nb)
            asm volatile(
                "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
                    "r"(st + (uint32_t)lane * a.lrow * 4), "l"(rows + (size_t)c * pitch + g0), "r"(nb), "r"(full)
                : "memory");
        asm volatile(
            "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
                "r"(st + data_bytes + (uint32_t)lane * T::WD * 4), "l"(desc + (size_t)c * descpitch + g_lo),
            "r"((uint32_t)T::WD * 4), "r"(full)
            : "memory");
        bytes = nb + T::WD * 4;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) bytes += __shfl_xor_sync(0xffffffffu, bytes, o);
    __syncwarp();  // the terminator row is written before lane 0's (releasing) arrive
    if (lane == 0)
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(full), "r"(bytes) : "memory");
}

// grid: min(tiles, SMs x CTAs per SM) persistent CTAs (tree_tile above).
template <typename T>
__global__ void __launch_bounds__(T::THREADS, T::MINB) tree_kernel(KArgs a, const uint32_t *desc,
                                                             int descpitch) {
    typedef typename T::Elem Elem;
    typedef typename T::Acc Acc;
    {
        uint64_t *full = reinterpret_cast<uint64_t *>(dedisp_smem);
        uint64_t *empty = full + T::NSTAGE;
        if (threadIdx.x == 0) {
            for (int s = 0; s < T::NSTAGE; ++s) {
                mbar_init(&full[s], 1);
                mbar_init(&empty[s], T::NW);
            }
            mbar_fence_init();
        }
        // the terminator descriptor row of every stage (row CC; never overwritten by the copies)
        const size_t sbytes = tree_stage_bytes<T>(a.lrow);
        if (threadIdx.x < T::NSTAGE * T::WD)
            reinterpret_cast<uint32_t *>(dedisp_smem + TreeSmem<T>::STAGES + (size_t)(threadIdx.x / T::WD) * sbytes +
                                         (size_t)T::CC * a.lrow * 4)[T::CC * T::WD + threadIdx.x % T::WD] = 0u;
    }
    __syncthreads();
    const int nchunks = (a.C + T::CC - 1) / T::CC;
    // prologue: warp 0 fills the first NSTAGE-1 stages
    constexpr int AHEAD = T::NSTAGE - 1;
    if (threadIdx.x < 32) {
        const int total = tree_my_tiles<T::PERSIST>(a) * nchunks;
        for (int g = 0; g < AHEAD && g < total; ++g) tree_issue<T>(a, desc, descpitch, g, nchunks);
    }

    Elem acc[T::DT][T::TT];
#pragma unroll
    for (int j = 0; j < T::DT; ++j)
#pragma unroll
        for (int k = 0; k < T::TT; ++k) acc[j][k] = 0;

    // Everything derived from the warp index -- the warp's DM group, its descriptors, every lattice
    // test -- is warp-uniform: the lattice branches never diverge.

    // uint8 input: add the 16-bit counters into the uint32 output (the first flush stores) and clear
    // them.  Every output element belongs to exactly one thread, so the read-modify-write needs no
    // atomics.  All loads of one (DM, half) are issued before the first add: TT/4 in flight.
    auto flush = [&](int it, bool first) {
        if constexpr (T::U8) {
            const uint32_t tid = sreg_tid();
            const int warp = tid >> 5, lane = tid & 31;
            int tx, ty, bz;
            tree_tile<T::PERSIST>(a, it, tx, ty, bz);
            const int dm0 = tx * T::DMS_CTA + (warp % T::WD) * T::DT;
            const int t0 = ty * T::HALF + (warp / T::WD) * 32 * T::TT + lane * T::TT;
            uint32_t *out = reinterpret_cast<uint32_t *>(a.out) + (size_t)bz * a.D * a.S;
            const bool vec = (a.S & 3) == 0;
#pragma unroll
            for (int j = 0; j < T::DT; ++j) {
                if (dm0 + j < a.D) {
                    uint32_t *o = out + (size_t)(dm0 + j) * a.S;
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        // low half: outputs t < S2; high half: outputs S2 + t < S
                        const int tb = h ? a.S2 + t0 : t0;
                        const int lim = h ? a.S : (a.S2 < a.S ? a.S2 : a.S);
                        if (vec && tb + T::TT <= lim) {
                            uint4 old[T::TT / 4];
                            if (!first) {
#pragma unroll
                                for (int k = 0; k < T::TT / 4; ++k)
                                    old[k] = *reinterpret_cast<const uint4 *>(o + tb + 4 * k);
                            } else {
#pragma unroll
                                for (int k = 0; k < T::TT / 4; ++k) old[k] = make_uint4(0, 0, 0, 0);
                            }
#pragma unroll
                            for (int k = 0; k < T::TT / 4; ++k) {
                                uint4 u = old[k];
                                if (h) {
                                    u.x += acc[j][4 * k] >> 16; u.y += acc[j][4 * k + 1] >> 16;
                                    u.z += acc[j][4 * k + 2] >> 16; u.w += acc[j][4 * k + 3] >> 16;
                                } else {
                                    u.x += acc[j][4 * k] & 0xffffu; u.y += acc[j][4 * k + 1] & 0xffffu;
                                    u.z += acc[j][4 * k + 2] & 0xffffu; u.w += acc[j][4 * k + 3] & 0xffffu;
                                }
                                *reinterpret_cast<uint4 *>(o + tb + 4 * k) = u;
                            }
                        } else {
#pragma unroll
                            for (int k = 0; k < T::TT; ++k)
                                if (tb + k < lim) {
                                    const uint32_t v = h ? acc[j][k] >> 16 : acc[j][k] & 0xffffu;
                                    o[tb + k] = first ? v : o[tb + k] + v;
                                }
                        }
                    }
                }
#pragma unroll
                for (int k = 0; k < T::TT; ++k) acc[j][k] = 0;
            }
        }
    };
    // What the channel loop keeps in registers besides the accumulators: the row pitch (an opaque move:
    // otherwise it is re-read from the constant bank in every channel).
    uint32_t lrow_b;
    asm volatile("mov.u32 %0, %1;" : "=r"(lrow_b) : "r"(a.lrow * 4));

    // One pass of the ring position g: wait for the chunk, add it, release its stage, and (one warp per
    // chunk, rotating: step a4) refill the most recently released stage with the chunk AHEAD positions on,
    // which may already belong to the CTA's next tile.
    auto ring_step = [&](int g) {
        const uint32_t s = g % T::NSTAGE;
        mbar_wait_s(smem_base() + TreeSmem<T>::FULL + s * 8, (g / T::NSTAGE) & 1);
        {
            // the thread's place in a staged row and the warp's descriptor column of this stage
            // (recomputed per chunk: two registers the channel loop does not have to spare)
            const uint32_t t = sreg_tid();
            const uint32_t warp = t >> 5, lane = t & 31;
            const uint32_t st = smem_base() + TreeSmem<T>::STAGES + s * (uint32_t)tree_stage_bytes<T>(a.lrow);
            const uint32_t my_row = st + ((warp / T::WD) * 32 * T::TT + lane * T::TT) * 4;
            const uint32_t my_desc = st + (uint32_t)T::CC * a.lrow * 4 + (warp % T::WD) * 4;
            TreeStep<Elem, T::DT, T::TT, T::QMAX, T::LAZY>::template chunk<T::WD>(acc, my_row, my_desc, lrow_b);
        }
        __syncwarp();
        const uint32_t tid = sreg_tid();
        if ((tid & 31) == 0) mbar_arrive_s(smem_base() + TreeSmem<T>::EMPTY + s * 8);
        const int gg = g + AHEAD;
        if ((int)(tid >> 5) == g % T::NW && gg < tree_my_tiles<T::PERSIST>(a) * nchunks) {
            if (gg >= T::NSTAGE)
                mbar_wait_s(smem_base() + TreeSmem<T>::EMPTY + (gg % T::NSTAGE) * 8, ((gg / T::NSTAGE) - 1) & 1);
            tree_issue<T>(a, desc, descpitch, gg, nchunks);
        }
    };

    if constexpr (T::U8) {
        // uint8: one tile per CTA (the launch makes the grid as large as the tile count; persistent CTAs
        // measured 1 % slower here).  The chunk loop runs in segments that end where this warp flushes its
        // counters: the flush sits OUTSIDE the inner loop, so that its register needs (20 registers of old
        // sums per DM half) do not make ptxas shuffle two dozen accumulators at every chunk's entry and exit.
        // The warps flush at different chunks (the others keep the pipes busy meanwhile): warp w after the
        // chunks k with (k + 1 + phase_w) a multiple of FLUSH_CHUNKS; no counter runs longer than
        // FLUSH_CHUNKS chunks (<= 256 channels) between two flushes.
        bool flushed = false;
        int k = 0;
        int kend = T::FLUSH_CHUNKS - ((int)(sreg_tid() >> 5) * T::FLUSH_CHUNKS) / T::NW;
        while (k < nchunks) {
            if (kend > nchunks) kend = nchunks;
#pragma unroll 1
            for (; k < kend; ++k) ring_step(k);
            if (k < nchunks) {
                flush(0, !flushed);
                flushed = true;
            }
            kend += T::FLUSH_CHUNKS;
        }
        flush(0, !flushed);   // step a6
    } else {
        // fp32: persistent CTAs; the ring runs on across the CTA's tiles, the store sits between them
        int g = 0;
        while (g < tree_my_tiles<T::PERSIST>(a) * nchunks) {
            const int gend = g + nchunks;
#pragma unroll 1
            for (; g < gend; ++g) ring_step(g);
            // store (step a6): each thread writes TT consecutive samples of each of its DMs
            const uint32_t tid = sreg_tid();
            const int warp = tid >> 5, lane = tid & 31;
            int tx, ty, bz;
            tree_tile<T::PERSIST>(a, g / nchunks - 1, tx, ty, bz);
            const int dm0 = tx * T::DMS_CTA + (warp % T::WD) * T::DT;
            const int t0 = ty * T::HALF + (warp / T::WD) * 32 * T::TT + lane * T::TT;
            Acc *out = (Acc *)a.out + (size_t)bz * a.D * a.S;
            const bool vec = (a.S & 3) == 0 && t0 + T::TT <= a.S;
#pragma unroll
            for (int j = 0; j < T::DT; ++j) {
                if (dm0 + j < a.D) {
                    float *o = out + (size_t)(dm0 + j) * a.S + t0;
                    if (vec) {
#pragma unroll
                        for (int k2 = 0; k2 < T::TT; k2 += 4)
                            *reinterpret_cast<float4 *>(o + k2) =
                                make_float4(acc[j][k2], acc[j][k2 + 1], acc[j][k2 + 2], acc[j][k2 + 3]);
                    } else {
#pragma unroll
                        for (int k2 = 0; k2 < T::TT; ++k2)
                            if (t0 + k2 < a.S) o[k2] = acc[j][k2];
                    }
                }
#pragma unroll
                for (int k2 = 0; k2 < T::TT; ++k2) acc[j][k2] = 0;
            }
        }
    }
}

}  // namespace dedisp

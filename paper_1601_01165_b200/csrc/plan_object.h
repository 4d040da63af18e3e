// plan_object.h -- the plan object behind the opaque dedisp_plan handle, and the host pipeline it owns.
// Included by the library's core translation units only (plan.cu, tuner.cu, host_pipe.cu,
// static_scratch.cu): the kernel variants never see a plan, so build.py does not rebuild them when
// this file changes.
#pragma once
#include "dedisp_internal.h"

namespace dedisp {

// Three-stage host pipeline of dedisp_execute_host_async (host_pipe.cu).
struct HostPipe {
    static constexpr int kSlots = 3;
    bool ready = false;
    cudaStream_t s_h2d = nullptr, s_exec = nullptr, s_d2h = nullptr;
    void *in[kSlots] = {}, *out[kSlots] = {};
    cudaEvent_t ev_in[kSlots] = {}, ev_exec[kSlots] = {}, ev_out[kSlots] = {};
    size_t in_bytes = 0, out_bytes = 0;
    uint64_t calls = 0;
    // streaming (dedisp_stream_block_async): what the LAST call left on the device, so that the block that
    // follows it in time takes its first M input columns from there instead of uploading them again
    bool st_valid = false;          // the last call was a stream block and its slot still holds its input
    const void *st_series = nullptr;
    int64_t st_pitch = 0, st_next_t0 = 0;
    int64_t st_h2d_bytes = 0;       // host-to-device bytes of the last stream block (DEDISP_STREAM_H2D_BYTES)
    void destroy();
};

}  // namespace dedisp

struct dedisp_plan {
    int C, D, dtype;
    int64_t S, M;
    int in_pitch, dpitch;
    double f_low, bw, rate, dm_first, dm_step;
    int32_t *d_shift = nullptr;
    int32_t *d_shiftT = nullptr;
    std::vector<int32_t> h_shift;  // [D][C]
    int max_step = 0;
    std::vector<dedisp::VariantFit> fit;  // per variant
    dedisp::TreeInfo tree;
    int variant = 0;
    int device = 0;                // the CUDA device the plan's tables live on
    int sm_count = 148;            // its SM count (the untuned default's wave quantisation)
    // uint8 tree kernels: the input repacked as pairs of samples S2 apart (pack_pairs_kernel)
    int S2 = 0, pair_pitch = 0;
    // The workspace is allocated when a tree_u8 variant is first selected (or by dedisp_plan_reserve) and
    // handed from stream to stream by an event: a call on another stream than the last one first makes
    // its stream wait for the last call's kernels (launch_variant).
    uint32_t *d_pairs = nullptr;   // [pairs_beams][C][pair_pitch]
    int pairs_beams = 0;
    std::vector<uint32_t *> retired_pairs;  // outgrown blocks: kernels in flight and captured graphs may
                                            // still name them, so they live until dedisp_plan_destroy
    mutable std::mutex pairs_mu;            // guards the four fields below and the enqueue of a paired call
    cudaEvent_t pairs_done = nullptr;       // recorded behind the last tree_u8 kernel that read d_pairs
    mutable cudaStream_t pairs_stream = nullptr;  // the stream of that call
    mutable bool pairs_used = false;
    // host-buffer path workspace (dedisp_execute_host)
    void *ws_in = nullptr, *ws_out = nullptr;
    size_t ws_in_bytes = 0, ws_out_bytes = 0;
    dedisp::HostPipe pipe;  // dedisp_execute_host_async
};

// static_scratch.cu -- dedisp_execute_static_scratch: the uint8 register-window path with its pair
// workspace in a fixed array that is part of the library image, for callers that must not (or cannot)
// allocate device memory.  Contract: include/dedisp.h.
//
// Who needs this.  dedisp_execute on a U8 plan reads the input through a workspace that
// dedisp_plan_create / dedisp_plan_reserve obtained with cudaMalloc.  Some code that wants to
// dedisperse has no way to get such a buffer:
//   - a process that has handed all free device memory to a pool (PyTorch's caching allocator, RMM):
//     a raw cudaMalloc fails there although the pool has room;
//   - a real-time block loop, where cudaMalloc / cudaFree serialise the whole device and stall the
//     other beams' streams for milliseconds;
//   - a thread that works while another thread captures a CUDA graph in the global capture mode,
//     where an allocation call is refused and breaks the capture.
// Such a caller takes a plan that set-up code created earlier (its tables are small) and calls the
// entry point below, which issues kernel launches and nothing else.
//
// The array lives in every CUDA context that loads this library, from module load to process exit,
// whether or not the entry point is ever called: kStaticScratchWords * 4 bytes per GPU.
#include <algorithm>
#include <cstdio>
#include <mutex>

#include "plan_object.h"

namespace dedisp {

// 4 Mi pair words = 16 MiB.  One beam needs nr_channels * PAIR_PITCH words (PAIR_PITCH is about
// nr_samples / 2 + max shift), so e.g. 256 channels x 16384 pairs fit; the survey-sized config
// (1536 channels x 44k pairs = 273 MB) does not and has to use dedisp_execute.
constexpr size_t kStaticScratchWords = (size_t)4 << 20;

// The scratch itself.  In DEVICE code this name is the array.  In HOST code the same name is only a
// handle the runtime uses to look the array up: it is not a device address, and a kernel handed
// `g_pair_scratch` from host code would fault, or, on a system where the GPU can reach host memory,
// quietly read and write some host bytes instead.  Host code therefore asks the runtime for the
// array's address on the current device (scratch_for_current_device) and passes that to the kernels.
static __device__ __align__(256) uint32_t g_pair_scratch[kStaticScratchWords];

constexpr int kMaxDevices = 64;
static std::mutex g_scratch_mu;
static uint32_t *g_scratch_ptr[kMaxDevices] = {};  // per device: the array's address there (0 = not asked yet)

// The array's device address on the CURRENT device.  Every device has its own copy of the array at
// its own address, so the address is looked up once per device, with that device current, and kept.
static int scratch_for_current_device(int dev, uint32_t **out) {
    if (dev < 0 || dev >= kMaxDevices) {
        set_last_error_text("dedisp_execute_static_scratch: device ordinal beyond the 64 this entry point tracks");
        return DEDISP_ERR_INVALID_ARG;
    }
    std::lock_guard<std::mutex> lk(g_scratch_mu);
    if (!g_scratch_ptr[dev]) {
        uint32_t *p = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void **)&p, g_pair_scratch);
        if (e != cudaSuccess || !p) {
            set_last_error("cudaGetSymbolAddress(static pair scratch)", e);
            return DEDISP_ERR_CUDA;
        }
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return DEDISP_OK;
}

}  // namespace dedisp

using namespace dedisp;

extern "C" {

int64_t dedisp_static_scratch_bytes(void) { return (int64_t)(kStaticScratchWords * sizeof(uint32_t)); }

int dedisp_execute_static_scratch(const dedisp_plan *plan, const void *d_in, void *d_out, int nr_beams,
                                  void *stream) {
    if (!plan || !d_in || !d_out || nr_beams < 1) return DEDISP_ERR_INVALID_ARG;
    if (((uintptr_t)d_in & 15) || ((uintptr_t)d_out & 15)) return DEDISP_ERR_INVALID_ARG;
    char msg[256];
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != plan->device) {
        snprintf(msg, sizeof msg, "the plan lives on device %d but the current device is %d", plan->device, dev);
        set_last_error_text(msg);
        return DEDISP_ERR_INVALID_ARG;
    }
    const Variant &x = variants()[plan->variant];
    if (plan->dtype != DEDISP_U8 || x.kind != KIND_TREE) {
        set_last_error_text("dedisp_execute_static_scratch: only U8 plans whose selected variant is a tree_u8 kernel "
                            "use scratch memory; call dedisp_execute, which needs none for this plan");
        return DEDISP_ERR_INVALID_ARG;
    }
    const TreeTable *tt = plan->tree.find_locked(x.dt, x.dms_cta);
    if (!tt) return DEDISP_ERR_INVALID_ARG;  // cannot happen for the selected variant: it was prepared
    const size_t beam_words = (size_t)plan->C * (size_t)plan->pair_pitch;
    if (beam_words > kStaticScratchWords) {
        snprintf(msg, sizeof msg,
                 "dedisp_execute_static_scratch: one beam needs %zu bytes of pair scratch (nr_channels %d x %d pairs "
                 "x 4), the static array holds %zu; use dedisp_execute",
                 beam_words * 4, plan->C, plan->pair_pitch, kStaticScratchWords * 4);
        set_last_error_text(msg);
        return DEDISP_ERR_INVALID_ARG;
    }
    uint32_t *scratch = nullptr;
    int rc = scratch_for_current_device(dev, &scratch);
    if (rc != DEDISP_OK) return rc;

    const VariantFit &f = plan->fit[plan->variant];
    KArgs a;
    a.shift = plan->d_shift; a.shiftT = plan->d_shiftT;
    a.C = plan->C; a.D = plan->D; a.S = (int)plan->S; a.in_pitch = plan->in_pitch;
    a.dpitch = plan->dpitch; a.lrow = f.lrow;
    a.pairs = scratch; a.pair_pitch = plan->pair_pitch; a.S2 = plan->S2;
    a.desc = tt->d_desc; a.descpitch = tt->pitch;
    a.nx = a.ny = a.ntiles = 0;  // filled in by the variant's launcher
    // As many beams per launch as the array holds; the groups follow each other on the stream, so a
    // group's packing kernel starts only after the previous group's add kernel has read the scratch.
    // Nothing in the scratch has to start at zero: the packing kernel rewrites every word the add
    // kernel can read (all pair_pitch words of every row of the group, zeros where a row has ended),
    // so what an earlier call left behind is never seen.
    const int group = (int)std::min<size_t>(kStaticScratchWords / beam_words, 65535);
    const size_t in_beam = (size_t)plan->C * plan->in_pitch;
    const size_t out_beam = (size_t)plan->D * plan->S * 4;
    cudaStream_t st = (cudaStream_t)stream;
    for (int b0 = 0; b0 < nr_beams; b0 += group) {
        const int nb = std::min(group, nr_beams - b0);
        a.in = (const char *)d_in + (size_t)b0 * in_beam;
        a.out = (char *)d_out + (size_t)b0 * out_beam;
        cudaError_t e = pack_pairs((const uint8_t *)a.in, scratch, nb, plan->C, plan->in_pitch, plan->pair_pitch,
                                   plan->S2, st);
        if (e == cudaSuccess) e = x.launch(a, nb, f.smem, st);
        if (e != cudaSuccess) { set_last_error(x.name, e); return DEDISP_ERR_CUDA; }
    }
    return DEDISP_OK;
}

}  // extern "C"

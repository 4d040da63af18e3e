// host_pipe.cu -- dedisp_execute_host_async / dedisp_host_sync: the end-to-end path for HOST buffers
// as a three-stage pipeline.  The paper keeps data resident on the device because dedispersion is
// one stage of a longer real-time pipeline; when the samples do come from
// the host, consecutive calls overlap: the H2D copy of call n+1, the kernel of call n and the D2H
// copy of call n-1 run on three streams over kSlots device workspaces, ordered by events.
#include <cstdio>

#include "plan_object.h"

using namespace dedisp;

extern "C" int dedisp_execute(const dedisp_plan *plan, const void *d_in, void *d_out, int nr_beams,
                              void *stream);

namespace dedisp {

void HostPipe::destroy() {
    for (int i = 0; i < kSlots; ++i) {
        if (in[i]) cudaFree(in[i]);
        if (out[i]) cudaFree(out[i]);
        if (ev_in[i]) cudaEventDestroy(ev_in[i]);
        if (ev_exec[i]) cudaEventDestroy(ev_exec[i]);
        if (ev_out[i]) cudaEventDestroy(ev_out[i]);
        in[i] = out[i] = nullptr;
        ev_in[i] = ev_exec[i] = ev_out[i] = nullptr;
    }
    if (s_h2d) cudaStreamDestroy(s_h2d);
    if (s_exec) cudaStreamDestroy(s_exec);
    if (s_d2h) cudaStreamDestroy(s_d2h);
    s_h2d = s_exec = s_d2h = nullptr;
    in_bytes = out_bytes = 0;
    ready = false;
    st_valid = false;
}

// Streams and events once; workspaces grown (after draining the pipeline) when a call needs more.
static int pipe_prepare(HostPipe &p, size_t in_bytes, size_t out_bytes) {
    cudaError_t e = cudaSuccess;
    if (!p.ready) {
        // a half-built pipeline is torn down again: the next call starts from scratch, nothing leaks
        if ((e = cudaStreamCreateWithFlags(&p.s_h2d, cudaStreamNonBlocking)) != cudaSuccess ||
            (e = cudaStreamCreateWithFlags(&p.s_exec, cudaStreamNonBlocking)) != cudaSuccess ||
            (e = cudaStreamCreateWithFlags(&p.s_d2h, cudaStreamNonBlocking)) != cudaSuccess) {
            set_last_error("cudaStreamCreate", e);
            p.destroy();
            return DEDISP_ERR_CUDA;
        }
        for (int i = 0; i < HostPipe::kSlots; ++i)
            if ((e = cudaEventCreateWithFlags(&p.ev_in[i], cudaEventDisableTiming)) != cudaSuccess ||
                (e = cudaEventCreateWithFlags(&p.ev_exec[i], cudaEventDisableTiming)) != cudaSuccess ||
                (e = cudaEventCreateWithFlags(&p.ev_out[i], cudaEventDisableTiming)) != cudaSuccess) {
                set_last_error("cudaEventCreate", e);
                p.destroy();
                return DEDISP_ERR_CUDA;
            }
        p.ready = true;
    }
    if (in_bytes > p.in_bytes || out_bytes > p.out_bytes) {
        cudaStreamSynchronize(p.s_h2d);
        cudaStreamSynchronize(p.s_exec);
        cudaStreamSynchronize(p.s_d2h);
        for (int i = 0; i < HostPipe::kSlots; ++i) {
            if (in_bytes > p.in_bytes) {
                if (p.in[i]) cudaFree(p.in[i]);
                p.in[i] = nullptr;
                if ((e = cudaMalloc(&p.in[i], in_bytes)) != cudaSuccess) break;
            }
            if (out_bytes > p.out_bytes) {
                if (p.out[i]) cudaFree(p.out[i]);
                p.out[i] = nullptr;
                if ((e = cudaMalloc(&p.out[i], out_bytes)) != cudaSuccess) break;
            }
        }
        if (e != cudaSuccess) {
            set_last_error("cudaMalloc(host pipeline workspace)", e);
            p.destroy();
            return DEDISP_ERR_ALLOC;
        }
        if (in_bytes > p.in_bytes) p.in_bytes = in_bytes;
        if (out_bytes > p.out_bytes) p.out_bytes = out_bytes;
        p.st_valid = false;  // the workspaces that held the last block are gone
    }
    return DEDISP_OK;
}

}  // namespace dedisp

#define PIPE_TRY(expr, what)                   \
    do {                                       \
        cudaError_t e_ = (expr);               \
        if (e_ != cudaSuccess) {               \
            set_last_error(what, e_);          \
            return DEDISP_ERR_CUDA;            \
        }                                      \
    } while (0)

// A failure in the middle of a pipelined call leaves copies and events of this slot enqueued without
// the ordering a later reuse of the slot relies on: drain the three streams before reporting it.
static int pipe_abort(dedisp::HostPipe &p, int rc) {
    cudaStreamSynchronize(p.s_h2d);
    cudaStreamSynchronize(p.s_exec);
    cudaStreamSynchronize(p.s_d2h);
    return rc;
}
#define PIPE_TRY_DRAIN(expr, what)             \
    do {                                       \
        cudaError_t e_ = (expr);               \
        if (e_ != cudaSuccess) {               \
            set_last_error(what, e_);          \
            return pipe_abort(p, DEDISP_ERR_CUDA); \
        }                                      \
    } while (0)

// One pipelined call.  series_pitch == 0: dense batch [nr_beams][C][in_pitch] -> [nr_beams][D][S].
// Otherwise one beam taken from / written to long host arrays: input rows of S+M samples at column
// t0 of rows series_pitch elements apart, output rows of S samples at column t0 of rows out_pitch
// elements apart (2-D copies).
static int pipe_call(dedisp_plan *plan, const void *h_in, void *h_out, int nr_beams,
                     int64_t series_pitch, int64_t out_pitch, int64_t t0) {
    const size_t esz = plan->dtype == DEDISP_U8 ? 1 : 4;
    const size_t in_bytes = (size_t)nr_beams * plan->C * plan->in_pitch * esz;
    const size_t out_bytes = (size_t)nr_beams * plan->D * plan->S * 4;
    HostPipe &p = plan->pipe;
    int rc = pipe_prepare(p, in_bytes, out_bytes);
    if (rc != DEDISP_OK) return rc;
    const int s = (int)(p.calls % HostPipe::kSlots);
    const bool reused = p.calls >= (uint64_t)HostPipe::kSlots;
    // stage 1: H2D into slot s once the kernel that last read this slot's input has finished
    if (reused) PIPE_TRY(cudaStreamWaitEvent(p.s_h2d, p.ev_exec[s], 0), "cudaStreamWaitEvent");
    if (series_pitch == 0) {
        p.st_valid = false;
        PIPE_TRY(cudaMemcpyAsync(p.in[s], h_in, in_bytes, cudaMemcpyHostToDevice, p.s_h2d), "H2D");
    } else {
        // Carry-over ("the last M input samples carried over"): if this block follows
        // the previous call's block in time on the same series, its input columns [t0, t0 + M) are the
        // columns [S, S + M) of the rows the previous call uploaded, which still sit in that call's slot.
        // They are moved device to device (on the upload stream, which ran that upload itself, so stream
        // order is enough), and only the S new columns of every row cross the bus.
        const bool carry = p.st_valid && p.st_series == h_in && p.st_pitch == series_pitch &&
                           p.st_next_t0 == t0 && p.calls > 0;
        p.st_valid = false;  // until this call has enqueued all of its copies
        const size_t row_bytes = (size_t)plan->in_pitch * esz;
        size_t skip = 0;     // leading columns of every row that do not come from the host
        if (carry && plan->M > 0) {
            const int prev = (int)((p.calls - 1) % HostPipe::kSlots);
            skip = (size_t)plan->M;
            PIPE_TRY_DRAIN(cudaMemcpy2DAsync(p.in[s], row_bytes, (const char *)p.in[prev] + (size_t)plan->S * esz,
                                             row_bytes, skip * esz, (size_t)plan->C, cudaMemcpyDeviceToDevice,
                                             p.s_h2d), "carry-over (D2D, 2-D)");
        }
        PIPE_TRY_DRAIN(cudaMemcpy2DAsync((char *)p.in[s] + skip * esz, row_bytes,
                                         (const char *)h_in + ((size_t)t0 + skip) * esz, (size_t)series_pitch * esz,
                                         ((size_t)(plan->S + plan->M) - skip) * esz, (size_t)plan->C,
                                         cudaMemcpyHostToDevice, p.s_h2d), "H2D (2-D)");
        p.st_h2d_bytes = (int64_t)(((size_t)(plan->S + plan->M) - skip) * esz * (size_t)plan->C);
    }
    PIPE_TRY_DRAIN(cudaEventRecord(p.ev_in[s], p.s_h2d), "cudaEventRecord");
    // stage 2: the kernels, once the input is there and the slot's previous output has left
    PIPE_TRY_DRAIN(cudaStreamWaitEvent(p.s_exec, p.ev_in[s], 0), "cudaStreamWaitEvent");
    if (reused) PIPE_TRY_DRAIN(cudaStreamWaitEvent(p.s_exec, p.ev_out[s], 0), "cudaStreamWaitEvent");
    rc = dedisp_execute(plan, p.in[s], p.out[s], nr_beams, p.s_exec);
    if (rc != DEDISP_OK) return pipe_abort(p, rc);
    PIPE_TRY_DRAIN(cudaEventRecord(p.ev_exec[s], p.s_exec), "cudaEventRecord");
    // stage 3: D2H
    PIPE_TRY_DRAIN(cudaStreamWaitEvent(p.s_d2h, p.ev_exec[s], 0), "cudaStreamWaitEvent");
    if (series_pitch == 0)
        PIPE_TRY_DRAIN(cudaMemcpyAsync(h_out, p.out[s], out_bytes, cudaMemcpyDeviceToHost, p.s_d2h), "D2H");
    else
        PIPE_TRY_DRAIN(cudaMemcpy2DAsync((char *)h_out + (size_t)t0 * 4, (size_t)out_pitch * 4, p.out[s],
                                   (size_t)plan->S * 4, (size_t)plan->S * 4, (size_t)plan->D,
                                   cudaMemcpyDeviceToHost, p.s_d2h), "D2H (2-D)");
    PIPE_TRY_DRAIN(cudaEventRecord(p.ev_out[s], p.s_d2h), "cudaEventRecord");
    ++p.calls;
    if (series_pitch != 0) {
        p.st_valid = true;
        p.st_series = h_in;
        p.st_pitch = series_pitch;
        p.st_next_t0 = t0 + plan->S;
    }
    return DEDISP_OK;
}

extern "C" int dedisp_execute_host_async(dedisp_plan *plan, const void *h_in, void *h_out,
                                         int nr_beams) {
    if (!plan || !h_in || !h_out || nr_beams < 1) return DEDISP_ERR_INVALID_ARG;
    return pipe_call(plan, h_in, h_out, nr_beams, 0, 0, 0);
}

extern "C" int dedisp_stream_block_async(dedisp_plan *plan, const void *h_series,
                                         int64_t series_pitch, void *h_out, int64_t out_pitch,
                                         int64_t t0) {
    if (!plan || !h_series || !h_out || t0 < 0 || series_pitch < t0 + plan->S + plan->M ||
        out_pitch < t0 + plan->S)
        return DEDISP_ERR_INVALID_ARG;
    return pipe_call(plan, h_series, h_out, 1, series_pitch, out_pitch, t0);
}

extern "C" int dedisp_stream_reset(dedisp_plan *plan) {
    if (!plan) return DEDISP_ERR_INVALID_ARG;
    plan->pipe.st_valid = false;
    return DEDISP_OK;
}

extern "C" int dedisp_host_sync(dedisp_plan *plan) {
    if (!plan) return DEDISP_ERR_INVALID_ARG;
    HostPipe &p = plan->pipe;
    if (!p.ready) return DEDISP_OK;
    PIPE_TRY(cudaStreamSynchronize(p.s_h2d), "cudaStreamSynchronize");
    PIPE_TRY(cudaStreamSynchronize(p.s_exec), "cudaStreamSynchronize");
    PIPE_TRY(cudaStreamSynchronize(p.s_d2h), "cudaStreamSynchronize");
    return DEDISP_OK;
}

// dedisp_internal.h -- plan object, kernel-argument block and the variant registry shared by the
// translation units of libdedisp_b200.so.  Not part of the public ABI (include/dedisp.h is).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <deque>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/dedisp.h"

namespace dedisp {

// Kernel families.
enum Kind {
    KIND_GENERIC = 0,  // one (DM, sample) per thread, global-memory reads (PAPER.md:173 baseline)
    KIND_LDS = 1,      // CTA tile staged in shared memory, one shared-memory word per add
    KIND_TREE = 3      // register window, offsets selected by a generated branch lattice
};

// Arguments every kernel receives by value.
struct KArgs {
    const void *in;          // [B][C][in_pitch]
    void *out;               // [B][D][S]
    const int32_t *shift;    // [D][C]          user-visible table
    const int32_t *shiftT;   // [C][dpitch]     transposed copy, DM axis padded with the last DM
    int C, D;
    int S;                   // output samples per beam
    int in_pitch;            // elements per input row (multiple of 16 bytes)
    int dpitch;              // ints per shiftT row (multiple of 128, >= D + 128)
    int lrow;                // shared-memory row pitch in staged elements (tiled kernels)
    const uint32_t *pairs;   // uint8 tree kernels: [B][C][pair_pitch] 16-bit sample pairs (workspace)
    int pair_pitch;          // pairs per row (multiple of 4)
    int S2;                  // pair y holds samples y and y + S2 (about S/2, multiple of 4)
    const uint32_t *desc;    // KIND_TREE: [C][descpitch] descriptors for the variant's tile
    int descpitch;
    int nx, ny, ntiles;      // KIND_TREE (persistent CTAs): DM tiles, time tiles, nx * ny * beams
};

// Per-variant numbers derived from the plan's shift table at plan creation.
struct VariantFit {
    bool ok = false;     // can run this plan
    int lrow = 0;        // shared-memory row pitch (elements)
    size_t smem = 0;     // dynamic shared memory bytes
    int span = 0;        // largest shift difference across one of the variant's DM tiles
};

struct PlanShape {
    int C, D, S, in_pitch, dtype;
    int S2;                  // uint8 pair layout: distance of the two samples of a pair
    int64_t M;               // max shift
    int max_step;            // max over (c,i) of shift(c,i+1)-shift(c,i)
    const int32_t *h_shift;  // host copy [D][C]
    const struct TreeInfo *tree;  // KIND_TREE tables
};

// Descriptor table of the KIND_TREE kernels for one (DT, DMs per CTA) pair, built by desc_kernel
// at plan creation.
struct TreeTable {
    int dt = 0, dms_cta = 0;
    uint32_t *d_desc = nullptr;  // [C][pitch]
    int pitch = 0;
};
struct TreeInfo {
    bool valid = false;  // every channel's increments are {q_c, q_c + 1}, q_c <= 7
    int qmax = -1;       // max_c q_c
    int *d_qc = nullptr; // device: q_c per channel
    mutable std::mutex mu;  // guards tables (built when a tree variant is first selected or run)
    std::deque<TreeTable> tables;  // a deque: push_back leaves the entries a launch has looked up in place
    const TreeTable *find(int dt, int dms_cta) const {   // caller holds mu
        for (const TreeTable &t : tables)
            if (t.dt == dt && t.dms_cta == dms_cta) return &t;
        return nullptr;
    }
    const TreeTable *find_locked(int dt, int dms_cta) const {
        std::lock_guard<std::mutex> lk(mu);
        return find(dt, dms_cta);
    }
};

struct Variant {
    const char *name;
    int dtype;        // DEDISP_F32 / DEDISP_U8
    int kind;
    int dms_cta;      // DMs per CTA
    int samples_cta;  // output samples per CTA
    int dt, tt;       // outputs per thread: dt DMs x tt samples
    int cc;           // channel-chunk depth (channels per pipeline stage)
    int stages;
    int qmax;         // KIND_TREE: largest slope class q_c the variant's lattice covers
    int lazy = 0;     // KIND_TREE: upper window quads loaded on demand (gen_tree.py)
    int threads;
    // Fills lrow/smem, returns whether the variant supports the plan.
    VariantFit (*fit)(const Variant &, const PlanShape &, int span_cta);
    cudaError_t (*launch)(const KArgs &, int nr_beams, size_t smem, cudaStream_t);
    cudaError_t (*prepare)(size_t smem);  // cudaFuncSetAttribute for large dynamic smem
};

// The registry: one entry per line of csrc/variants.py, in that order (build/registry_gen.inc).
const std::vector<Variant> &variants();

// shift_table.cu
cudaError_t build_shift_tables(int C, double f_low, double bw, double rate, double dm_first,
                               double dm_step, int D, int dpitch, int32_t *d_shift,
                               int32_t *d_shiftT, int *d_flag, cudaStream_t st);

cudaError_t build_chan_slopes(const int32_t *d_shiftT, int C, int D, int dpitch, int *d_qc,
                              int *d_flags, cudaStream_t st);
cudaError_t build_tree_desc(const int32_t *d_shiftT, const int *d_qc, int C, int D, int dpitch,
                            int dt, int dms_cta, int al, int descpitch, uint32_t *d_desc,
                            int *d_flags, cudaStream_t st);

cudaError_t pack_pairs(const uint8_t *d_in, uint32_t *d_pairs, int nr_beams, int C, int in_pitch,
                       int pair_pitch, int S2, cudaStream_t st);

void set_last_error(const char *what, cudaError_t e);
void set_last_error_text(const char *msg);  // a message that is not a CUDA error (dedisp_last_error)

}  // namespace dedisp

// shift_table.cu -- steps a1-a3: trial DMs, channel frequencies and the int32
// shift table Delta(chan, dm) of Eq. (1), computed on the device in IEEE
// double with the fixed association of DESIGN.md reading A3.  Every operation is an explicit
// round-to-nearest intrinsic so that ptxas cannot contract a multiply and an add into an FMA.
#include "dedisp_internal.h"

namespace dedisp {

__device__ __forceinline__ double delay_samples(double f, double f_h, double dm, double rate) {
    double a = __ddiv_rn(1.0, __dmul_rn(f, f));
    double b = __ddiv_rn(1.0, __dmul_rn(f_h, f_h));
    double diff = __dsub_rn(a, b);
    double k = __dmul_rn(__dmul_rn(4150.0, dm), diff);  // Eq. (1): seconds
    return __dmul_rn(k, rate);
}

// One thread per (dm i, channel c).  Writes shift[i][c] and shiftT[c][i]; DM-axis padding of
// shiftT (i in [D, dpitch)) repeats the last DM so that ragged DM tiles read in-bounds spans.
__global__ void shift_table_kernel(int C, double f_low, double bw, double rate, double dm_first,
                                   double dm_step, int D, int dpitch, int32_t *shift,
                                   int32_t *shiftT, int *flag) {
    int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= C) return;
    for (int i = blockIdx.y; i < dpitch; i += gridDim.y) {
    int ii = i < D ? i : D - 1;
    double f = __dadd_rn(f_low, __dmul_rn((double)c, bw));    // reading A1: f_c = f_low + c*bw
    double f_h = __dadd_rn(f_low, __dmul_rn((double)C, bw));  // band top edge
    double dm = __dadd_rn(dm_first, __dmul_rn((double)ii, dm_step));  // reading A5
    double x = delay_samples(f, f_h, dm, rate);
    double fl = floor(x);
    // reading A4: nearest, ties up (x >= 0).  x - fl is exact.
    double r = fl + ((__dsub_rn(x, fl) >= 0.5) ? 1.0 : 0.0);
    int32_t s;
    if (!(r >= 0.0) || !(r <= 2147483647.0)) {
        atomicOr(flag, 1);
        s = 0;
    } else {
        s = (int32_t)r;
    }
    if (i < D) shift[(size_t)i * C + c] = s;
    shiftT[(size_t)c * dpitch + i] = s;
    }
}

cudaError_t build_shift_tables(int C, double f_low, double bw, double rate, double dm_first,
                               double dm_step, int D, int dpitch, int32_t *d_shift,
                               int32_t *d_shiftT, int *d_flag, cudaStream_t st) {
    dim3 block(128);
    dim3 grid((C + 127) / 128, dpitch < 65535 ? dpitch : 65535);
    shift_table_kernel<<<grid, block, 0, st>>>(C, f_low, bw, rate, dm_first, dm_step, D, dpitch,
                                               d_shift, d_shiftT, d_flag);
    return cudaGetLastError();
}

// KIND_TREE tables (kernel_tree.cuh).
// chan_slope_kernel: one block per channel c.  q_c = min over i of shift(c,i+1) - shift(c,i); the
// tree kernels need every increment of the channel to be q_c or q_c + 1 (true for a rounded linear
// function of the DM index).  flags[0] = max_c q_c, flags[1] = 1 if some channel violates it.
__global__ void chan_slope_kernel(const int32_t *shiftT, int D, int dpitch, int *qc, int *flags) {
    const int c = blockIdx.x;
    const int32_t *row = shiftT + (size_t)c * dpitch;
    int mn = 0x7fffffff, mx = 0;
    for (int i = threadIdx.x; i + 1 < D; i += blockDim.x) {
        int d = row[i + 1] - row[i];
        mn = d < mn ? d : mn;
        mx = d > mx ? d : mx;
    }
    __shared__ int smn[128], smx[128];
    smn[threadIdx.x] = mn;
    smx[threadIdx.x] = mx;
    __syncthreads();
    for (int o = 64; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
            smn[threadIdx.x] = min(smn[threadIdx.x], smn[threadIdx.x + o]);
            smx[threadIdx.x] = max(smx[threadIdx.x], smx[threadIdx.x + o]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        mn = smn[0];
        mx = smx[0];
        if (mn == 0x7fffffff) mn = 0;  // D == 1
        if (mn < 0 || mn > 7 || mx - mn > 1) {
            atomicOr(&flags[1], 1);
            mn = 0;
        }
        atomicMax(&flags[0], mn);
        qc[c] = mn;
    }
}

// desc_kernel: one thread per (channel c, DM group G of dt DMs); the group belongs to the CTA tile
// of dms_cta DMs that starts at DM lo = (G*dt / dms_cta) * dms_cta.  With
//   woff = shift(c, G*dt) - (shift(c, lo) & ~(al-1)): offset of the group's first DM in the staged
//          row, whose element 0 is row element T0 + (shift(c, lo) & ~(al-1)),
//   desc[c][G] = bits << 24 | (0x10000 << q_c) | (woff >> 2) << 4 | (woff & 3)      (gen_tree.py)
// i.e. d & 0xfff0 is the byte offset of the 16-byte quad the window starts in, d & 3 the first DM's
// offset in it, and increment j of the group = q_c + bit (j-1)  (dt <= 9, q_c <= 7).
// DMs past D (ragged last group, padding groups) continue with increment q_c: their outputs are
// never stored and their window offsets stay inside the lattice.  flags[1] |= 1 if woff >= 2^14.
__global__ void desc_kernel(const int32_t *shiftT, const int *qc, int C, int D, int dpitch, int dt,
                            int dms_cta, int al, int descpitch, uint32_t *desc, int *flags) {
    int G = blockIdx.x * blockDim.x + threadIdx.x;
    int c = blockIdx.y;
    if (G >= descpitch) return;
    const int32_t *row = shiftT + (size_t)c * dpitch;
    const long d0 = (long)G * dt;
    const long lo = d0 / dms_cta * dms_cta;
    const int e0 = row[d0 < D ? d0 : D - 1];
    const int base = row[lo < D ? lo : D - 1] & ~(al - 1);  // al = staged elements per 16 bytes
    const int q = qc[c];
    uint32_t bits = 0;
    for (int j = 1; j < dt && d0 + j < D; ++j) {
        int b = (row[d0 + j] - row[d0 + j - 1]) - q;
        b = b < 0 ? 0 : b > 1 ? 1 : b;  // only when flags[1] is already set
        bits |= (uint32_t)b << (j - 1);
    }
    const int woff = e0 - base;
    if (woff < 0 || woff > 0x3fff) atomicOr(&flags[1], 1);
    const uint32_t w = (uint32_t)woff & 0x3fffu;
    desc[(size_t)c * descpitch + G] = bits << 24 | (0x10000u << q) | (w >> 2) << 4 | (w & 3u);
}

// pack_pairs_kernel: the uint8 tree kernels' view of the input (kernel_tree.cuh).  One thread per four
// pairs: pairs[b][c][y] = in[b][c][y] | in[b][c][y + S2] << 16, samples past the row read as 0.
__global__ void pack_pairs_kernel(const uint8_t *in, uint32_t *pairs, int in_pitch, int pair_pitch,
                                  int S2) {
    const int y4 = blockIdx.x * blockDim.x + threadIdx.x;  // group of four pairs
    if (4 * y4 >= pair_pitch) return;
    const size_t row = blockIdx.y + (size_t)blockIdx.z * gridDim.y;
    const uint32_t *r = reinterpret_cast<const uint32_t *>(in + row * in_pitch);
    const int n4 = in_pitch >> 2;  // in_pitch is a multiple of 16
    const uint32_t lo = y4 < n4 ? r[y4] : 0u;
    const uint32_t hi = y4 + (S2 >> 2) < n4 ? r[y4 + (S2 >> 2)] : 0u;
    const uint32_t le = __byte_perm(lo, 0, 0x4240), lq = __byte_perm(lo, 0, 0x4341);
    const uint32_t he = __byte_perm(hi, 0, 0x4240), hq = __byte_perm(hi, 0, 0x4341);
    uint4 v;
    v.x = __byte_perm(le, he, 0x5410);
    v.y = __byte_perm(lq, hq, 0x5410);
    v.z = __byte_perm(le, he, 0x7632);
    v.w = __byte_perm(lq, hq, 0x7632);
    reinterpret_cast<uint4 *>(pairs + row * pair_pitch)[y4] = v;
}

cudaError_t pack_pairs(const uint8_t *d_in, uint32_t *d_pairs, int nr_beams, int C, int in_pitch,
                       int pair_pitch, int S2, cudaStream_t st) {
    dim3 block(256);
    dim3 grid((pair_pitch / 4 + 255) / 256, C, nr_beams);
    pack_pairs_kernel<<<grid, block, 0, st>>>(d_in, d_pairs, in_pitch, pair_pitch, S2);
    return cudaGetLastError();
}

cudaError_t build_chan_slopes(const int32_t *d_shiftT, int C, int D, int dpitch, int *d_qc,
                              int *d_flags, cudaStream_t st) {
    chan_slope_kernel<<<C, 128, 0, st>>>(d_shiftT, D, dpitch, d_qc, d_flags);
    return cudaGetLastError();
}

cudaError_t build_tree_desc(const int32_t *d_shiftT, const int *d_qc, int C, int D, int dpitch,
                            int dt, int dms_cta, int al, int descpitch, uint32_t *d_desc,
                            int *d_flags, cudaStream_t st) {
    dim3 block(128);
    dim3 grid((descpitch + 127) / 128, C);
    desc_kernel<<<grid, block, 0, st>>>(d_shiftT, d_qc, C, D, dpitch, dt, dms_cta, al, descpitch,
                                        d_desc, d_flags);
    return cudaGetLastError();
}

}  // namespace dedisp

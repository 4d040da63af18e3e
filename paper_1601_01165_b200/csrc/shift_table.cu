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

}  // namespace dedisp

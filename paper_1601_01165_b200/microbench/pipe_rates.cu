// pipe_rates.cu -- the microbenchmarks behind DESIGN.md section 6: issue rates of the plain ALU pipes
// (FADD, packed FADD2, integer adds, DP4A, PRMT, LOP3, IMAD), shared-memory bandwidth per access width,
// shared-memory loads mixed with FADDs, and the cost of warp-uniform two-way branches between short
// FADD blocks.  Measurement only; not part of libdedisp_b200.so.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o pipe_rates pipe_rates.cu && ./pipe_rates
// Every number is per SM: lane-operations (or bytes) per SM clock, from clock64() spans taken over all
// warps of one CTA per SM (148 CTAs).
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>

#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("CUDA %s at %d\n", cudaGetErrorString(e), __LINE__); return 1; } } while (0)

constexpr int NACC = 16;
constexpr int ITERS = 4096;
#define TEND __shared__ unsigned long long tmin, tmax; if (threadIdx.x == 0) { tmin = ~0ull; tmax = 0; } __syncthreads(); \
    atomicMin(&tmin, (unsigned long long)t0); atomicMax(&tmax, (unsigned long long)t1); __syncthreads();

// mode: 0 FADD, 1 FADD2, 2 IADD (2-in), 3 IADD3, 4 FADD+IADD3 1:1, 5 FFMA, 6 dp4a, 7 PRMT, 8 LOP3, 9 IMAD,
// 10 FADD + IADD3 2:1, 11 FADD with same src (reg bank), 12 FADD2+IADD3 1:1
template <int MODE>
__global__ void __launch_bounds__(1024) k_alu(const float *src, float *dst, long long *cyc) {
    float a[NACC], x[NACC];
    unsigned ia[NACC], ix[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) {
        a[i] = src[threadIdx.x + i * 32];
        x[i] = src[threadIdx.x + 1024 + i * 32];
        ia[i] = __float_as_uint(a[i]);
        ix[i] = __float_as_uint(x[i]);
    }
    __syncthreads();
    long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < ITERS; ++it) {
#pragma unroll
        for (int i = 0; i < NACC; ++i) {
            if (MODE == 0) asm volatile("add.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(x[i]));
            if (MODE == 11) asm volatile("add.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(x[0]));
            if (MODE == 1 || MODE == 12) {
                if (i % 2 == 0)
                    asm volatile("{.reg .b64 p, q; mov.b64 p, {%0, %1}; mov.b64 q, {%2, %3}; add.f32x2 p, p, q; mov.b64 {%0, %1}, p;}"
                                 : "+f"(a[i]), "+f"(a[i + 1]) : "f"(x[i]), "f"(x[i + 1]));
            }
            if (MODE == 2) asm volatile("add.u32 %0, %0, %1;" : "+r"(ia[i]) : "r"(ix[i]));
            if (MODE == 3) asm volatile("{.reg .u32 t; add.u32 t, %1, %2; add.u32 %0, %0, t;}" : "+r"(ia[i]) : "r"(ix[i]), "r"(ix[(i + 1) % NACC]));
            if (MODE == 4 || MODE == 10) {
                asm volatile("add.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(x[i]));
                if (MODE == 4 || (i % 2 == 0))
                    asm volatile("{.reg .u32 t; add.u32 t, %1, %2; add.u32 %0, %0, t;}" : "+r"(ia[i]) : "r"(ix[i]), "r"(ix[(i + 1) % NACC]));
            }
            if (MODE == 12) asm volatile("{.reg .u32 t; add.u32 t, %1, %2; add.u32 %0, %0, t;}" : "+r"(ia[i]) : "r"(ix[i]), "r"(ix[(i + 1) % NACC]));
            if (MODE == 5) asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(a[i]) : "f"(x[i]), "f"(x[(i + 1) % NACC]));
            if (MODE == 6) asm volatile("dp4a.u32.u32 %0, %1, %2, %0;" : "+r"(ia[i]) : "r"(ix[i]), "r"(ix[(i + 1) % NACC]));
            if (MODE == 7) asm volatile("prmt.b32 %0, %0, %1, %2;" : "+r"(ia[i]) : "r"(ix[i]), "r"(ix[(i + 1) % NACC]));
            if (MODE == 8) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(ia[i]) : "r"(ix[i]), "r"(ix[(i + 1) % NACC]));
            if (MODE == 9) asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(ia[i]) : "r"(ix[i]), "r"(ix[(i + 1) % NACC]));
        }
    }
    long long t1 = clock64();
    TEND
    float s = 0;
    unsigned u = 0;
#pragma unroll
    for (int i = 0; i < NACC; ++i) { s += a[i]; u += ia[i]; }
    dst[blockIdx.x * blockDim.x + threadIdx.x] = s + __uint_as_float(u);
    if (threadIdx.x == 0) cyc[blockIdx.x] = tmax - tmin;
}

// LDS bandwidth: W = words per load (1,2,4). Optional NF FADDs per loaded word set.
template <int W, int NF>
__global__ void __launch_bounds__(1024) k_lds(const float *src, float *dst, long long *cyc) {
    extern __shared__ float sm[];
    for (int i = threadIdx.x; i < 8192; i += blockDim.x) sm[i] = src[i % 2048];
    __syncthreads();
    float acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    float f[NF > 0 ? NF : 1];
    for (int i = 0; i < NF; ++i) f[i] = 0;
    int base = (threadIdx.x * W) & 4095;
    long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < ITERS; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            int off = (base + u * 256 * W / 4 * 4 + (it & 3) * 4) & 8191 & ~(W - 1);
            if (W == 1) { float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"((unsigned)__cvta_generic_to_shared(sm + off))); acc[u] += v; }
            if (W == 2) { float v, w; asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(v), "=f"(w) : "r"((unsigned)__cvta_generic_to_shared(sm + off))); acc[u] += v + w; }
            if (W == 4) { float v, w, y, z; asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v), "=f"(w), "=f"(y), "=f"(z) : "r"((unsigned)__cvta_generic_to_shared(sm + off))); acc[u] += (v + w) + (y + z); }
#pragma unroll
            for (int i = 0; i < NF; ++i) asm volatile("add.f32 %0, %0, %1;" : "+f"(f[i]) : "f"(acc[u]));
        }
    }
    long long t1 = clock64();
    TEND
    float s = 0;
    for (int u = 0; u < 8; ++u) s += acc[u];
    for (int i = 0; i < NF; ++i) s += f[i];
    dst[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0) cyc[blockIdx.x] = tmax - tmin;
}

// uniform branch cost: each iteration executes NB blocks of 8 FADDs; before each block a warp-uniform
// two-way branch selects one of two equivalent blocks depending on bits of a loaded word.
template <int NB>
__global__ void __launch_bounds__(1024) k_branch(const float *src, const unsigned *bits, float *dst, long long *cyc) {
    float a[8], x[10];
    for (int i = 0; i < 8; ++i) a[i] = src[threadIdx.x + i * 32];
    for (int i = 0; i < 10; ++i) x[i] = src[threadIdx.x + 512 + i * 32];
    __shared__ unsigned sb[256];
    if (threadIdx.x < 256) sb[threadIdx.x] = bits[threadIdx.x];
    __syncthreads();
    long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < ITERS; ++it) {
        unsigned b = __shfl_sync(0xffffffffu, sb[(it + (threadIdx.x >> 5)) & 255], 0);
#pragma unroll
        for (int j = 0; j < NB; ++j) {
            if (b & (1u << j)) {
#pragma unroll
                for (int i = 0; i < 8; ++i) asm volatile("add.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(x[i + 1]));
            } else {
#pragma unroll
                for (int i = 0; i < 8; ++i) asm volatile("add.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(x[i]));
            }
        }
    }
    long long t1 = clock64();
    TEND
    float s = 0;
    for (int i = 0; i < 8; ++i) s += a[i];
    dst[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0) cyc[blockIdx.x] = tmax - tmin;
}

static float *d_src, *d_dst;
static unsigned *d_bits;
static long long *d_cyc;

template <typename F>
static double run(F launch, int blocks) {
    launch();
    cudaDeviceSynchronize();
    launch();
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) { printf("err %s\n", cudaGetErrorString(e)); return -1; }
    static long long h[4096];
    cudaMemcpy(h, d_cyc, blocks * sizeof(long long), cudaMemcpyDeviceToHost);
    double m = 0;
    for (int i = 0; i < blocks; ++i) m += h[i];
    return m / blocks;
}

int main() {
    CK(cudaMalloc(&d_src, 1 << 20));
    CK(cudaMalloc(&d_dst, 148 * 8 * 1024 * 4));
    CK(cudaMalloc(&d_cyc, 4096 * 8));
    CK(cudaMalloc(&d_bits, 1024));
    static float h[1 << 18];
    for (int i = 0; i < (1 << 18); ++i) h[i] = (float)(i % 7) * 1e-3f;
    CK(cudaMemcpy(d_src, h, 1 << 20, cudaMemcpyHostToDevice));
    unsigned hb[256];
    unsigned s = 12345;
    for (int i = 0; i < 256; ++i) { s = s * 1664525u + 1013904223u; hb[i] = s >> 8; }
    CK(cudaMemcpy(d_bits, hb, 1024, cudaMemcpyHostToDevice));
    const int blocks = 148;
    const char *names[] = {"FADD", "FADD2(f32x2)", "IADD", "IADD3", "FADD+IADD3 1:1", "FFMA", "DP4A", "PRMT", "LOP3", "IMAD", "FADD+IADD3 2:1", "FADD samesrc", "FADD2+IADD3"};
    // ops per thread per iter (counting lane-ops: adds)
    const double ops[] = {NACC, NACC, NACC, 2 * NACC, 3 * NACC, NACC, NACC, NACC, NACC, NACC, 2 * NACC, NACC, 3 * NACC};
    for (int threads : {256, 512, 1024}) {
#define RUN(M) { double c = run([&] { k_alu<M><<<blocks, threads>>>(d_src, d_dst, d_cyc); }, blocks); \
        printf("%-16s thr %4d: %8.1f lane-ops/clk/SM  (%.2f cyc/iter)\n", names[M], threads, ops[M] * ITERS * threads / c, c / ITERS); }
        RUN(0) RUN(1) RUN(2) RUN(3) RUN(4) RUN(5) RUN(6) RUN(7) RUN(8) RUN(9) RUN(10) RUN(11) RUN(12)
    }
    for (int threads : {256, 512, 1024}) {
#define RUNL(W, NF) { cudaFuncSetAttribute(k_lds<W, NF>, cudaFuncAttributeMaxDynamicSharedMemorySize, 32768); \
        double c = run([&] { k_lds<W, NF><<<blocks, threads, 32768>>>(d_src, d_dst, d_cyc); }, blocks); \
        printf("LDS.%d +%d FADD/ld thr %4d: %7.1f B/clk/SM, %7.1f FADD/clk/SM\n", W * 32, NF, threads, 8.0 * W * 4 * ITERS * threads / c, 8.0 * NF * ITERS * threads / c); }
        RUNL(1, 0) RUNL(2, 0) RUNL(4, 0) RUNL(4, 8) RUNL(4, 12) RUNL(4, 16) RUNL(1, 2) RUNL(1, 3)
    }
    for (int threads : {256, 512}) {
#define RUNB(NB) { double c = run([&] { k_branch<NB><<<blocks, threads>>>(d_src, d_bits, d_dst, d_cyc); }, blocks); \
        printf("branch NB=%d thr %4d: %7.1f FADD/clk/SM (%.1f cyc/iter/warp-slot)\n", NB, threads, 8.0 * NB * ITERS * threads / c, c / ITERS); }
        RUNB(1) RUNB(4) RUNB(8)
    }
    return 0;
}

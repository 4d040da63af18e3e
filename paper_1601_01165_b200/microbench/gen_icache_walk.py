"""gen_icache_walk.py -- instruction-cache microbenchmark behind DESIGN.md section 7: a warp-uniform random
walk over NB straight-line blocks of NF FADDs (one two-way branch per block), for code footprints from 3.5 KB
to 56 KB.  Writes icache_walk.cu; build and run:
    python gen_icache_walk.py 20 8 48 64 80 96 112 128
    nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o icache_walk icache_walk.cu && ./icache_walk
"""
import sys
NF=int(sys.argv[1]); sizes=[int(x) for x in sys.argv[2:]]
o=[]
o.append('#include <cstdio>\n#include <cuda_runtime.h>\n')
o.append('__device__ __forceinline__ void blk(float (&a)[%d], const float (&x)[%d], int r){\n' % (NF, NF+4))
o.append('#pragma unroll\n for(int k=0;k<%d;++k) asm volatile("add.f32 %%0, %%0, %%1;" : "+f"(a[k]) : "f"(x[k+(r&3)]));\n}\n' % NF)
for NB in sizes:
    o.append('__global__ void __launch_bounds__(1024) walk%d(const float* src, float* dst, long long* cyc, int steps, unsigned seed){\n' % NB)
    o.append(' float a[%d], x[%d]; for(int i=0;i<%d;++i) a[i]=src[threadIdx.x+i]; for(int i=0;i<%d;++i) x[i]=src[threadIdx.x+64+i];\n' % (NF,NF+4,NF,NF+4))
    o.append(' unsigned s = seed + 977u*(threadIdx.x>>5) + 131u*blockIdx.x; s = __shfl_sync(0xffffffffu, s, 0); int n=0; unsigned bits=(s>>8)|0x1000000u;\n')
    o.append(' __syncthreads(); long long t0=clock64();\n goto B0;\n')
    import random
    rnd=random.Random(NB)
    for b in range(NB):
        s0=rnd.randrange(NB); s1=rnd.randrange(NB)
        o.append(' B%d: blk(a,x,%d); bits>>=1; if(bits==1u){ n+=24; if(n>=steps) goto DONE; s=s*1664525u+1013904223u; bits=(s>>8)|0x1000000u; } if(bits&1) goto B%d; else goto B%d;\n' % (b,b,s0,s1))
    o.append(' DONE: long long t1=clock64(); __shared__ unsigned long long tmin,tmax; if(threadIdx.x==0){tmin=~0ull;tmax=0;} __syncthreads(); atomicMin(&tmin,(unsigned long long)t0); atomicMax(&tmax,(unsigned long long)t1); __syncthreads();\n')
    o.append(' float r=0; for(int i=0;i<%d;++i) r+=a[i]; dst[blockIdx.x*blockDim.x+threadIdx.x]=r; if(threadIdx.x==0) cyc[blockIdx.x]=tmax-tmin;\n}\n' % NF)
o.append('int main(){ float *src,*dst; long long* cyc; cudaMalloc(&src,1<<20); cudaMemset(src,0,1<<20); cudaMalloc(&dst,148*1024*4); cudaMalloc(&cyc,148*8); const int steps=24000; long long h[148];\n')
for NB in sizes:
    o.append(' for(int thr: {128,256,384,512}){ for(int rep=0;rep<2;++rep){ walk%d<<<148,thr>>>(src,dst,cyc,steps,1234u); cudaDeviceSynchronize(); } cudaMemcpy(h,cyc,148*8,cudaMemcpyDeviceToHost); double m=0; for(int i=0;i<148;++i) m+=h[i]; m/=148; printf("NF=%d NB=%%4d (%%6.1f KB) thr %%4d: %%6.1f cyc/block/warp-slot, %%6.1f FADD/clk/SM\\n", %d, %d*(%d+8)*16/1024.0, thr, m/steps, (double)steps*%d*thr/m); }\n' % (NB,NF,NB,NB,NF,NF))
o.append(' return 0; }\n')
open('icache_walk.cu','w').write(''.join(o))

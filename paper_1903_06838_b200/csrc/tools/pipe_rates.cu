// pipe_rates.cu — issue-rate micro-benchmark behind DESIGN.md §5.1: cycles per instruction group and SM sub-partition
// for single instruction classes and pairs (which pipes overlap).  Not part of libpdp.so.
// Build + run: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -o pipe_rates pipe_rates.cu && ./pipe_rates
#include <cstdio>
#include <cuda_runtime.h>
#include <stdint.h>
#define ITER 1024
#define BENCH_KERNEL(name, BODY)                                                \
  __global__ void name(unsigned *out, long long *cyc, unsigned seed) {          \
    unsigned a0=seed,a1=seed+1,a2=seed+2,a3=seed+3,a4=seed+4,a5=seed+5,a6=seed+6,a7=seed+7; \
    unsigned c0=seed*3,c1=seed*3+1,c2=seed*3+2,c3=seed*3+3,c4=seed*3+4,c5=seed*3+5,c6=seed*3+6,c7=seed*3+7; \
    unsigned b = seed * 7u + threadIdx.x, c = seed * 5u + 7u;                   \
    __shared__ uint4 sm[1024];                                                  \
    sm[threadIdx.x] = make_uint4(b, c, b, c);                                   \
    __syncthreads();                                                            \
    long long t0 = clock64();                                                   \
    _Pragma("unroll 1") for (int it = 0; it < ITER; ++it) { BODY(0) BODY(1) BODY(2) BODY(3) BODY(4) BODY(5) BODY(6) BODY(7) } \
    long long t1 = clock64();                                                   \
    __syncthreads();                                                            \
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;                            \
    out[blockIdx.x * blockDim.x + threadIdx.x] = a0+a1+a2+a3+a4+a5+a6+a7+c0+c1+c2+c3+c4+c5+c6+c7; \
  }
#define FFMA(i) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+r"(a##i) : "r"(b), "r"(c));
#define FFMA_C(i) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+r"(c##i) : "r"(b), "r"(c));
#define PRMT(i) asm volatile("prmt.b32 %0, %0, %1, 0x6240;" : "+r"(c##i) : "r"(b));
#define LOP3(i) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(c##i) : "r"(b), "r"(c));
#define HFMA2(i) asm volatile("fma.rn.f16x2 %0, %0, %1, %2;" : "+r"(c##i) : "r"(b), "r"(c));
#define HFMA2_A(i) asm volatile("fma.rn.f16x2 %0, %0, %1, %2;" : "+r"(a##i) : "r"(b), "r"(c));
#define FSET(i) asm volatile("set.lt.f32.f32 %0, %0, %1;" : "+r"(c##i) : "r"(b));
#define FSET_A(i) asm volatile("set.lt.f32.f32 %0, %0, %1;" : "+r"(a##i) : "r"(b));
#define HSET2(i) asm volatile("set.lt.f16x2.f16x2 %0, %0, %1;" : "+r"(c##i) : "r"(b));
#define FSETPSEL(i) asm volatile("{.reg .pred p; setp.lt.f32 p, %0, %1; selp.b32 %0, %1, %2, p;}" : "+r"(c##i) : "r"(b), "r"(c));
#define FMNMX(i) asm volatile("min.f32 %0, %0, %1;" : "+r"(c##i) : "r"(b));
#define IADD(i) asm volatile("add.u32 %0, %0, %1;" : "+r"(c##i) : "r"(b));
#define I2F(i) asm volatile("cvt.rn.f32.u32 %0, %0;" : "+r"(c##i));
#define F2FP(i) asm volatile("cvt.rn.f16x2.f32 %0, %0, %1;" : "+r"(c##i) : "r"(b));
#define LDS128(i) { uint4 v; asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x),"=r"(v.y),"=r"(v.z),"=r"(v.w) : "r"((unsigned)__cvta_generic_to_shared(&sm[(threadIdx.x + i * 32) & 1023]))); c##i ^= v.x ^ v.y ^ v.z ^ v.w; }
#define LDS32(i) { unsigned v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"((unsigned)__cvta_generic_to_shared(&sm[(threadIdx.x + i*32)&1023]))); c##i ^= v; }
#define SHFL(i) asm volatile("shfl.sync.bfly.b32 %0, %0, 1, 0x1f, 0xffffffff;" : "+r"(c##i));
#define VOTE(i) asm volatile("{.reg .pred p; setp.ne.u32 p, %0, 0; vote.sync.ballot.b32 %0, p, 0xffffffff;}" : "+r"(c##i));

#define P1(i) FFMA(i)
BENCH_KERNEL(k_ffma, P1)
#define P2(i) FFMA(i) FFMA_C(i)
BENCH_KERNEL(k_ffma2, P2)
#define P3(i) FFMA(i) PRMT(i)
BENCH_KERNEL(k_ffma_prmt, P3)
#define P4(i) FFMA(i) HFMA2(i)
BENCH_KERNEL(k_ffma_hfma2, P4)
#define P5(i) HFMA2_A(i) PRMT(i)
BENCH_KERNEL(k_hfma2_prmt, P5)
#define P6(i) FSET(i)
BENCH_KERNEL(k_fset, P6)
#define P7(i) FFMA(i) FSET(i)
BENCH_KERNEL(k_ffma_fset, P7)
#define P8(i) FSET_A(i) PRMT(i)
BENCH_KERNEL(k_fset_prmt, P8)
#define P9(i) HSET2(i)
BENCH_KERNEL(k_hset2, P9)
#define P10(i) HFMA2_A(i) HSET2(i)
BENCH_KERNEL(k_hfma2_hset2, P10)
#define P11(i) FSETPSEL(i)
BENCH_KERNEL(k_fsetp_sel, P11)
#define P12(i) FFMA(i) FMNMX(i)
BENCH_KERNEL(k_ffma_fmnmx, P12)
#define P13(i) FFMA(i) IADD(i)
BENCH_KERNEL(k_ffma_iadd, P13)
#define P14(i) I2F(i)
BENCH_KERNEL(k_i2f, P14)
#define P15(i) FFMA(i) I2F(i)
BENCH_KERNEL(k_ffma_i2f, P15)
#define P16(i) PRMT(i) 
BENCH_KERNEL(k_prmt, P16)
#define P17(i) FFMA(i) FFMA_C(i) PRMT(i)
BENCH_KERNEL(k_ffma2_prmt, P17)
#define P18(i) LDS128(i)
BENCH_KERNEL(k_lds128_xor2, P18)
#define P19(i) LDS32(i)
BENCH_KERNEL(k_lds32_xor, P19)
#define P20(i) FFMA(i) SHFL(i)
BENCH_KERNEL(k_ffma_shfl, P20)
#define P21(i) FFMA(i) VOTE(i)
BENCH_KERNEL(k_ffma_setp_vote, P21)
#define P22(i) FFMA(i) F2FP(i)
BENCH_KERNEL(k_ffma_f2fp, P22)
#define P23(i) FFMA(i) FFMA_C(i) HFMA2(i)
BENCH_KERNEL(k_ffma2_hfma2, P23)
#define P24(i) HFMA2_A(i) FSET(i)
BENCH_KERNEL(k_hfma2_fset, P24)
#define P25(i) FFMA(i) FSETPSEL(i)
BENCH_KERNEL(k_ffma_fsetp_sel, P25)

typedef void (*kfn)(unsigned *, long long *, unsigned);
struct Entry { const char *name; kfn fn; int n; };
int main() {
  Entry es[] = {{"ffma", k_ffma, 1}, {"ffma+ffma", k_ffma2, 2}, {"ffma+prmt", k_ffma_prmt, 2}, {"ffma+hfma2", k_ffma_hfma2, 2},
                {"hfma2+prmt", k_hfma2_prmt, 2}, {"fset", k_fset, 1}, {"ffma+fset", k_ffma_fset, 2}, {"fset+prmt", k_fset_prmt, 2},
                {"hset2", k_hset2, 1}, {"hfma2+hset2", k_hfma2_hset2, 2}, {"fsetp+sel", k_fsetp_sel, 2}, {"ffma+fmnmx", k_ffma_fmnmx, 2},
                {"ffma+iadd", k_ffma_iadd, 2}, {"i2f", k_i2f, 1}, {"ffma+i2f", k_ffma_i2f, 2}, {"prmt", k_prmt, 1},
                {"ffma+ffma+prmt", k_ffma2_prmt, 3}, {"lds128+2lop3", k_lds128_xor2, 3}, {"lds32+lop", k_lds32_xor, 2},
                {"ffma+shfl", k_ffma_shfl, 2}, {"ffma+setp+vote", k_ffma_setp_vote, 3}, {"ffma+f2fp", k_ffma_f2fp, 2},
                {"ffma+ffma+hfma2", k_ffma2_hfma2, 3}, {"hfma2+fset", k_hfma2_fset, 2}, {"ffma+fsetp+sel", k_ffma_fsetp_sel, 3}};
  unsigned *out; long long *cyc;
  cudaMalloc(&out, 148 * 1024 * 4); cudaMalloc(&cyc, 148 * 8);
  for (int threads : {512, 1024}) {
    printf("threads/CTA=%d (warps per SMSP=%d)\n", threads, threads / 128);
    for (auto &e : es) {
      e.fn<<<148, threads>>>(out, cyc, 1u);
      e.fn<<<148, threads>>>(out, cyc, 1u);
      cudaDeviceSynchronize();
      long long h[148]; cudaMemcpy(h, cyc, sizeof(h), cudaMemcpyDeviceToHost);
      double avg = 0; for (int i = 0; i < 148; ++i) avg += h[i]; avg /= 148;
      double groups = (double)(threads / 128) * ITER * 8;  // per SMSP
      printf("  %-18s cycles/group/SMSP=%.3f  (n=%d instr per group; + 3/8 loop instr)\n", e.name, avg / groups, e.n);
    }
  }
  printf("status: %s\n", cudaGetErrorString(cudaGetLastError()));
  return 0;
}

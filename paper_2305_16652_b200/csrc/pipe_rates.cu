// pipe_rates.cu — debug target, NOT part of libhcc_b200.so: the issue rate of each instruction class the
// encoder (encode.cu) and the traversal kernel (trace.cu) are made of, measured on the GPU it runs on.
// DESIGN.md §6 bounds both kernels by instruction issue, not by HBM; the rates it quotes come from here
// (profiles/r3_pipe_rates.md holds the table and the command).
//
//   python -m paper_2305_16652_b200.build --pipe-rates      # nvcc ... -o paper_2305_16652_b200/pipe_rates
//   ./paper_2305_16652_b200/pipe_rates
//
// Method: one CTA of 1,024 threads per SM (8 warps per scheduler), every thread runs CHAINS independent
// dependency chains of one instruction (inline PTX, so the compiler can neither merge nor drop them), ITERS
// times; the CTA's cycles are read with clock64 around the loop.  rate = warp-instructions issued per
// scheduler and clock = ITERS * CHAINS * (warps per scheduler) / cycles.  A "pair" row interleaves two
// classes one to one and reports the rate of the SUM: 1.0 there with 0.5 for each alone means the two
// dual-issue on different pipes.  Loop overhead (one add, one compare, one branch per ITER of 64+
// instructions) is below 3 %.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

#define CHAINS 8
#define UNROLL 8

enum Op {
    OP_FFMA, OP_FADD, OP_FMUL, OP_FMNMX, OP_FMNMX3, OP_PRMT, OP_LOP3, OP_FSEL, OP_FSETP_SEL, OP_IADD, OP_IMAD, OP_IMAD_HI,
    OP_FADD2, OP_FMUL2, OP_FFMA2, OP_PAIR_FFMA_PRMT, OP_PAIR_FFMA_FMNMX, OP_PAIR_FFMA_IMAD, OP_PAIR_FMNMX_PRMT, OP_PAIR_FADD2_FMNMX3,
    OP_COUNT
};
static const char *OP_NAME[OP_COUNT] = {
    "FFMA (fma.rn.f32)", "FADD (add.f32)", "FMUL (mul.f32)", "FMNMX (min.f32, 2 inputs)", "FMNMX3 (min.f32, 3 inputs)",
    "PRMT (prmt.b32)", "LOP3 (lop3.b32)", "ISETP + FSEL (setp.ne.u32 ; selp.f32), both", "FSETP + SEL (setp.lt.f32 ; selp.b32), both",
    "IADD3 (add.u32)", "IMAD (mad.lo.u32)", "IMAD.HI (mul.hi.u32)", "FADD2 (add.rn.f32x2)", "FMUL2 (mul.rn.f32x2)",
    "FFMA2 (fma.rn.f32x2)", "pair FFMA + PRMT", "pair FFMA + FMNMX", "pair FFMA + IMAD", "pair FMNMX + PRMT", "pair FADD2 + FMNMX3"};
// instructions issued per chain step (a pair row issues two)
static const int OP_WIDTH[OP_COUNT] = {1, 1, 1, 1, 1, 1, 1, 2, 2, 1, 1, 1, 1, 1, 1, 2, 2, 2, 2, 2};

template <int OP>
__device__ __forceinline__ void step(float &f, uint32_t &u, unsigned long long &d, float a, float b, uint32_t ua, uint32_t ub,
                                     unsigned long long da, float &g, uint32_t &v) {
    if (OP == OP_FFMA) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f) : "f"(a), "f"(b));
    if (OP == OP_FADD) asm volatile("add.f32 %0, %0, %1;" : "+f"(f) : "f"(a));
    if (OP == OP_FMUL) asm volatile("mul.f32 %0, %0, %1;" : "+f"(f) : "f"(a));
    if (OP == OP_FMNMX) asm volatile("min.f32 %0, %0, %1;" : "+f"(f) : "f"(a));
    if (OP == OP_FMNMX3) asm volatile("min.f32 %0, %0, %1, %2;" : "+f"(f) : "f"(a), "f"(b));
    if (OP == OP_PRMT) asm volatile("prmt.b32 %0, %0, %1, %2;" : "+r"(u) : "r"(ua), "r"(ub));
    if (OP == OP_LOP3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(u) : "r"(ua), "r"(ub));
    if (OP == OP_FSEL) asm volatile("{ .reg .pred p; setp.ne.u32 p, %2, 0; selp.f32 %0, %0, %1, p; }" : "+f"(f) : "f"(a), "r"(ua));
    if (OP == OP_FSETP_SEL) asm volatile("{ .reg .pred p; setp.lt.f32 p, %2, %3; selp.b32 %0, %0, %1, p; }" : "+r"(u) : "r"(ua), "f"(f), "f"(a));
    if (OP == OP_IADD) asm volatile("add.u32 %0, %0, %1;" : "+r"(u) : "r"(ua));
    if (OP == OP_IMAD) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(u) : "r"(ua), "r"(ub));
    if (OP == OP_IMAD_HI) asm volatile("mul.hi.u32 %0, %0, %1;" : "+r"(u) : "r"(ua));
    if (OP == OP_FADD2) asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(d) : "l"(da));
    if (OP == OP_FMUL2) asm volatile("mul.rn.f32x2 %0, %0, %1;" : "+l"(d) : "l"(da));
    if (OP == OP_FFMA2) asm volatile("fma.rn.f32x2 %0, %0, %1, %1;" : "+l"(d) : "l"(da));
    if (OP == OP_PAIR_FFMA_PRMT) {
        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f) : "f"(a), "f"(b));
        asm volatile("prmt.b32 %0, %0, %1, %2;" : "+r"(u) : "r"(ua), "r"(ub));
    }
    if (OP == OP_PAIR_FFMA_FMNMX) {
        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f) : "f"(a), "f"(b));
        asm volatile("min.f32 %0, %0, %1;" : "+f"(g) : "f"(a));
    }
    if (OP == OP_PAIR_FFMA_IMAD) {
        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f) : "f"(a), "f"(b));
        asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(u) : "r"(ua), "r"(ub));
    }
    if (OP == OP_PAIR_FMNMX_PRMT) {
        asm volatile("min.f32 %0, %0, %1;" : "+f"(f) : "f"(a));
        asm volatile("prmt.b32 %0, %0, %1, %2;" : "+r"(u) : "r"(ua), "r"(ub));
    }
    if (OP == OP_PAIR_FADD2_FMNMX3) {
        asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(d) : "l"(da));
        asm volatile("min.f32 %0, %0, %1, %2;" : "+f"(f) : "f"(a), "f"(b));
    }
    (void)v;
}

template <int OP>
__global__ void __launch_bounds__(1024, 1) k_rate(int iters, const float *in, float *sink, unsigned long long *cycles) {
    float f[CHAINS], g[CHAINS];
    uint32_t u[CHAINS], v[CHAINS];
    unsigned long long d[CHAINS];
    const float a = in[0], b = in[1];                     // run-time values: nothing folds
    const uint32_t ua = __float_as_uint(in[2]) | 1u, ub = __float_as_uint(in[3]) & 0x7777u;
    const unsigned long long da = ((unsigned long long)__float_as_uint(in[1]) << 32) | __float_as_uint(in[0]);
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) {
        f[c] = in[4] + (float)(threadIdx.x + c);
        g[c] = f[c] * 0.5f;
        u[c] = threadIdx.x * 2654435761u + c;
        v[c] = u[c] ^ 0x55u;
        d[c] = ((unsigned long long)__float_as_uint(f[c]) << 32) | __float_as_uint(g[c]);
    }
    __syncthreads();
    const long long t0 = clock64();
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < UNROLL; ++r)
#pragma unroll
            for (int c = 0; c < CHAINS; ++c) step<OP>(f[c], u[c], d[c], a, b, ua, ub, da, g[c], v[c]);
    }
    __syncthreads();
    const long long t1 = clock64();
    float acc = 0.f;
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) acc += f[c] + g[c] + (float)(u[c] ^ v[c]) + (float)(d[c] >> 40);
    if (acc == 1.2345e-30f) sink[0] = acc;                // keeps every chain alive
    if (threadIdx.x == 0) cycles[blockIdx.x] = (unsigned long long)(t1 - t0);
}

typedef void (*kern_t)(int, const float *, float *, unsigned long long *);
template <int OP> struct Table { static void fill(kern_t *t) { t[OP] = k_rate<OP>; Table<OP + 1>::fill(t); } };
template <> struct Table<OP_COUNT> { static void fill(kern_t *) {} };

int main(int argc, char **argv) {
    int iters = 4096, dev = 0;
    if (argc > 1) iters = atoi(argv[1]);
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) { fprintf(stderr, "no CUDA device\n"); return 1; }
    const int sms = prop.multiProcessorCount;
    float h_in[8] = {1.0000001f, 1e-9f, 3.0f, 5.0f, 0.25f, 0, 0, 0};
    float *d_in, *d_sink;
    unsigned long long *d_cyc, *h_cyc = new unsigned long long[sms];
    cudaMalloc(&d_in, sizeof(h_in)); cudaMalloc(&d_sink, 64); cudaMalloc(&d_cyc, sizeof(unsigned long long) * sms);
    cudaMemcpy(d_in, h_in, sizeof(h_in), cudaMemcpyHostToDevice);
    kern_t table[OP_COUNT];
    Table<0>::fill(table);
    printf("# %s, %d SMs, %d iterations x %d chains x %d unrolled, 1 CTA of 1024 threads per SM (8 warps per scheduler)\n",
           prop.name, sms, iters, CHAINS, UNROLL);
    printf("%-48s %14s %22s\n", "instruction class", "cycles (max)", "warp-instr/sched/clk");
    for (int op = 0; op < OP_COUNT; ++op) {
        table[op]<<<sms, 1024>>>(iters / 8, d_in, d_sink, d_cyc);      // warm-up
        table[op]<<<sms, 1024>>>(iters, d_in, d_sink, d_cyc);
        if (cudaDeviceSynchronize() != cudaSuccess) { fprintf(stderr, "kernel %d failed: %s\n", op, cudaGetErrorString(cudaGetLastError())); return 1; }
        cudaMemcpy(h_cyc, d_cyc, sizeof(unsigned long long) * sms, cudaMemcpyDeviceToHost);
        unsigned long long mx = 0;
        for (int i = 0; i < sms; ++i) mx = h_cyc[i] > mx ? h_cyc[i] : mx;
        const double instr = (double)iters * UNROLL * CHAINS * OP_WIDTH[op] * 8.0;    // per scheduler: 8 warps
        printf("%-48s %14llu %22.3f\n", OP_NAME[op], mx, instr / (double)mx);
    }
    return 0;
}

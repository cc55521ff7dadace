// pipe_rates.cu -- stand-alone microbenchmark behind DESIGN.md's ALU roofline denominators: thread-instructions per
// clock per SM of the instruction kinds the raster and the convolution lean on (FFMA, packed FFMA2/FADD2, DFMA/DADD/
// DMUL, the IMAD.WIDE + LOP3 pair of a Philox round) and the rate of RED.ADD.F32 into an S-sized grid.
// Built by `python -m paper_2203_02479_b200.build --pipe-rates` into paper_2203_02479_b200/pipe_rates; not part of
// libwcsim.so and not on the hot path.
#include <cstdio>
#include <cuda_runtime.h>
#include <stdint.h>

#define ITERS 4096
#define CHAINS 8

template <int KIND>
__global__ void __launch_bounds__(256) k(float *out, float a, float b, double da, double db, unsigned ua)
{
    float x[CHAINS];
    float2 x2[CHAINS];
    double d[CHAINS];
    unsigned u[CHAINS];
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) {
        x[c] = threadIdx.x * 1e-3f + c;
        x2[c] = make_float2(x[c], x[c] + 1.f);
        d[c] = x[c];
        u[c] = threadIdx.x + c;
    }
    const float2 a2 = make_float2(a, a * 0.5f), b2 = make_float2(b, b * 0.5f);
    // per-thread register operands (read from memory so they are not constant-bank or uniform operands)
    float y[CHAINS], z[CHAINS];
    float2 y2[CHAINS], z2[CHAINS];
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) {
        y[c] = out[(threadIdx.x + c) & 3] + 1.0f;
        z[c] = out[(threadIdx.x + 2 * c) & 3] + 0.5f;
        y2[c] = make_float2(y[c], z[c]);
        z2[c] = make_float2(z[c], y[c]);
    }
    for (int it = 0; it < ITERS; ++it) {
#pragma unroll
        for (int c = 0; c < CHAINS; ++c) {
            if (KIND == 0) x[c] = fmaf(x[c], a, b);
            if (KIND == 1) x2[c] = __ffma2_rn(x2[c], a2, b2);
            if (KIND == 2) x[c] = x[c] + a;
            if (KIND == 3) x2[c] = __fadd2_rn(x2[c], a2);
            if (KIND == 4) x2[c] = __fmul2_rn(x2[c], a2);
            if (KIND == 5) d[c] = fma(d[c], da, db);
            if (KIND == 6) d[c] = d[c] + da;
            if (KIND == 7) { // philox-like: mul.wide + xor
                unsigned long long p = (unsigned long long)u[c] * 0xD2511F53ull;
                u[c] = (unsigned)(p >> 32) ^ (unsigned)p ^ ua;
            }
            if (KIND == 8) { // FFMA + FADD mix (two pipes?)
                x[c] = fmaf(x[c], a, b);
                x2[c].x = x2[c].x + a;
            }
            if (KIND == 9) x[c] = x[c] * a;
            if (KIND == 10) { // FFMA2 + FADD mix
                x2[c] = __ffma2_rn(x2[c], a2, b2);
                x[c] = x[c] + a;
            }
            if (KIND == 11) d[c] = d[c] * da;
            if (KIND == 12) x[c] = fmaf(y[c], z[c], x[c]);
            if (KIND == 13) x[c] = x[c] + y[c];
            if (KIND == 14) x2[c] = __ffma2_rn(y2[c], z2[c], x2[c]);
            if (KIND == 15) x[c] = x[c] * y[c];
            if (KIND == 16) x2[c] = __fadd2_rn(x2[c], y2[c]);
        }
    }
    float s = 0;
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) s += x[c] + x2[c].x + x2[c].y + (float)d[c] + (float)u[c];
    if (s == 123.456f) out[0] = s;
}

// RED throughput: each warp adds to 32 consecutive floats at a pseudo-random row; MODE 0 distinct per warp, 1 all warps same line
template <int MODE>
__global__ void red_k(float *S, int n_lines, int iters)
{
    unsigned w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    unsigned h = w * 2654435761u;
    for (int i = 0; i < iters; ++i) {
        h = h * 1664525u + 1013904223u;
        unsigned line = MODE == 0 ? (h >> 8) % n_lines : (MODE == 1 ? 0 : (w * 7 + i / 30) % n_lines);
        atomicAdd(S + (size_t)line * 32 + lane, 1.0f);
    }
}

template <int KIND>
void run(const char *name, double ops_per_inner)
{
    float *out;
    cudaMalloc(&out, 16);
    cudaMemset(out, 0, 16);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int ctas = 148 * 8;
    k<KIND><<<ctas, 256>>>(out, 1.0001f, 0.5f, 1.0001, 0.5, 77u);
    cudaEventRecord(e0);
    k<KIND><<<ctas, 256>>>(out, 1.0001f, 0.5f, 1.0001, 0.5, 77u);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms;
    cudaEventElapsedTime(&ms, e0, e1);
    const double inst = (double)ctas * 256 * ITERS * CHAINS * ops_per_inner; // thread-level instructions
    int clk;
    cudaDeviceGetAttribute(&clk, cudaDevAttrClockRate, 0);
    const double cycles = ms * 1e-3 * clk * 1e3;
    printf("%-22s %8.3f ms  %7.1f thread-inst/clk/SM  (%.2f Tinst/s)\n", name, ms, inst / cycles / 148.0, inst / ms * 1e-9);
    cudaFree(out);
}

int main()
{
    run<0>("FFMA 3-reg", 1);
    run<12>("FFMA 3 distinct regs", 1);
    run<1>("FFMA2", 1);
    run<14>("FFMA2 3 distinct regs", 1);
    run<13>("FADD reg+reg", 1);
    run<15>("FMUL reg*reg", 1);
    run<16>("FADD2 reg+reg", 1);
    run<2>("FADD", 1);
    run<3>("FADD2", 1);
    run<4>("FMUL2", 1);
    run<9>("FMUL", 1);
    run<5>("DFMA", 1);
    run<6>("DADD", 1);
    run<11>("DMUL", 1);
    run<7>("IMAD.WIDE+LOP3 (x2)", 2);
    run<8>("FFMA+FADD mix (x2)", 2);
    run<10>("FFMA2+FADD mix (x2)", 2);
    // RED
    float *S;
    const int n_lines = 800 * 6000 / 32;
    cudaMalloc(&S, (size_t)n_lines * 128);
    cudaMemset(S, 0, (size_t)n_lines * 128);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    for (int mode = 0; mode < 3; ++mode) {
        const int ctas = 148 * 8, iters = 256;
        for (int rep = 0; rep < 2; ++rep) {
            cudaEventRecord(e0);
            if (mode == 0) red_k<0><<<ctas, 256>>>(S, n_lines, iters);
            if (mode == 1) red_k<1><<<ctas, 256>>>(S, n_lines, iters);
            if (mode == 2) red_k<2><<<ctas, 256>>>(S, n_lines, iters);
            cudaEventRecord(e1);
            cudaEventSynchronize(e1);
        }
        float ms;
        cudaEventElapsedTime(&ms, e0, e1);
        const double reds = (double)ctas * 256 * iters;
        printf("RED.ADD.F32 mode %d (0 random lines, 1 one line, 2 track-like): %.3f ms, %.1f G lane-adds/s, %.2f G warp-reds/s\n", mode, ms,
               reds / ms * 1e-6, reds / 32 / ms * 1e-6);
    }
    printf("err %s\n", cudaGetErrorString(cudaDeviceSynchronize()));
    return 0;
}

// unit_rates.cu -- stand-alone micro-benchmark of the per-SM instruction rates DESIGN.md section 7 builds its roofline on.
// Not part of libtpcf.so.  Build and run on the B200 box:
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/unit_rates paper_1204_6630_b200/csrc/unit_rates.cu && /tmp/unit_rates
// Every kernel runs the same shape: one CTA of 1024 threads per SM (32 warps, 8 per scheduler), each thread 8 independent
// dependency chains of one instruction kind, kIters x 8 instructions; rate = lane-instructions / (SM clocks elapsed),
// clocks from clock64() of the slowest CTA.  Output: one line per instruction kind, lanes per clock per SM.
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <vector>

constexpr int kIters = 4096, kThreads = 1024, kChains = 8;

#define CHECK(x)                                                                              \
    do {                                                                                      \
        cudaError_t e_ = (x);                                                                 \
        if (e_ != cudaSuccess) { std::fprintf(stderr, "%s: %s\n", #x, cudaGetErrorString(e_)); std::exit(1); } \
    } while (0)

template <int KIND>
__global__ void __launch_bounds__(kThreads) rate_kernel(float seed, float* sink, long long* clocks) {
    __shared__ unsigned hist[4096];
    __shared__ float4 row[32];
    for (int k = threadIdx.x; k < 4096; k += kThreads) hist[k] = 0;
    if (threadIdx.x < 32) row[threadIdx.x] = make_float4(seed, seed + 1.f, seed + 2.f, seed + 3.f);
    float a[kChains], b = seed * 1.0001f, c = seed * 0.5f;
    unsigned u[kChains];
    double d[kChains];
    unsigned long long p[kChains];
#pragma unroll
    for (int k = 0; k < kChains; ++k) {
        a[k] = seed + k + threadIdx.x;
        u[k] = threadIdx.x * 2654435761u + k;
        d[k] = seed + k;
        p[k] = ((unsigned long long)__float_as_uint(a[k]) << 32) | u[k];
    }
    __syncthreads();
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
        for (int k = 0; k < kChains; ++k) {
            if (KIND == 0) a[k] = fmaf(a[k], b, c);                                                        // FFMA
            if (KIND == 1) a[k] = a[k] + b;                                                                // FADD
            if (KIND == 2) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p[k]) : "l"(p[(k + 1) & 7]), "l"(p[(k + 2) & 7]));   // FFMA2, 2 FMA per lane
            if (KIND == 3) u[k] = (u[k] ^ (u[k] >> 3)) & 0x7FFFFC;                                          // LOP3 (+ SHF): ALU pipe
            if (KIND == 4) a[k] = fminf(fminf(a[k], b), c + (float)it);                                     // FMNMX / FMNMX3
            if (KIND == 5) u[k] = __umulhi(u[k], 0x9E3779B9u) + 1u;                                         // IMAD.HI
            if (KIND == 6) d[k] = fma(d[k], 1.0000001, 0.5);                                                // DFMA
            if (KIND == 7) { atomicAdd(&hist[(u[k] >> 7) & 4095], 1u); u[k] += 0x2000u * 37u; }             // ATOMS.POPC.INC, scattered words
            if (KIND == 8) atomicAdd(&hist[k], 1u);                                                         // ATOMS.POPC.INC, one word per warp instruction
            if (KIND == 9) { const float4 r = row[(it + k) & 31]; a[k] += (r.x + r.y) + (r.z + r.w); }        // broadcast LDS.128 (+ 3 FADD)
        }
    }
    const long long t1 = clock64();
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kChains; ++k) s += a[k] + (float)u[k] + (float)d[k] + (float)(p[k] & 0xFFFF);
    if (s == 12345.678f) sink[0] = s + hist[threadIdx.x];
    if (threadIdx.x == 0) clocks[blockIdx.x] = t1 - t0;
}

template <int KIND>
static void run(const char* name, double per_inst, int sms, float* sink, long long* dclk) {
    std::vector<long long> h(sms);
    rate_kernel<KIND><<<sms, kThreads>>>(1.5f, sink, dclk);      // warm-up
    rate_kernel<KIND><<<sms, kThreads>>>(1.5f, sink, dclk);
    CHECK(cudaDeviceSynchronize());
    CHECK(cudaMemcpy(h.data(), dclk, sms * sizeof(long long), cudaMemcpyDeviceToHost));
    long long worst = 0;
    for (long long v : h) worst = v > worst ? v : worst;
    const double lanes = (double)kIters * kChains * kThreads * per_inst;
    std::printf("%-58s %8.1f lanes/clk/SM  (%lld clk)\n", name, lanes / (double)worst, worst);
}

int main() {
    int sms = 0;
    CHECK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0));
    float* sink;
    long long* dclk;
    CHECK(cudaMalloc(&sink, 4096));
    CHECK(cudaMalloc(&dclk, sms * sizeof(long long)));
    std::printf("SMs %d; one CTA of %d threads per SM, %d chains x %d iterations per thread\n", sms, kThreads, kChains, kIters);
    run<0>("FFMA", 1, sms, sink, dclk);
    run<1>("FADD", 1, sms, sink, dclk);
    run<2>("FFMA2 (fma.rn.f32x2), counted as 2 FMA per lane", 2, sms, sink, dclk);
    run<3>("LOP3 + SHF pair (ALU pipe), counted as 2", 2, sms, sink, dclk);
    run<4>("FMNMX x2 / FMNMX3 (+ the loop's I2F/FADD), counted as 1", 1, sms, sink, dclk);
    run<5>("IMAD.HI (+ IADD)", 1, sms, sink, dclk);
    run<6>("DFMA", 1, sms, sink, dclk);
    run<7>("ATOMS.POPC.INC, lanes scattered over 4096 words", 1, sms, sink, dclk);
    run<8>("ATOMS.POPC.INC, all 32 lanes on one word", 1, sms, sink, dclk);
    run<9>("broadcast LDS.128 (+ 3 FADD), counted per load", 1, sms, sink, dclk);
    return 0;
}

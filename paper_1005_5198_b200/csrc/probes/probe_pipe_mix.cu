// probe_pipe_mix.cu -- issue-slot / register-bandwidth probe behind DESIGN.md section 5 ("Roofline").
//
// Not part of the library: a stand-alone microbenchmark that measures, on the GPU it runs on, how many cycles an
// SM sub-partition needs for a stream of packed FFMA2 (three operand patterns), scalar FADD and MUFU.RCP in the ratio
// of the shoot kernel's inner loop (40 FFMA2-class + 4 FADD + 0..12 MUFU per lens and thread), at 3 and 4 warps per
// scheduler.  Its output is committed as profiles/r01_probe_pipe_mix.txt.
//
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -o /tmp/probe_pipe_mix \
//        paper_1005_5198_b200/csrc/probes/probe_pipe_mix.cu && /tmp/probe_pipe_mix
//
// form 0: acc = fma2(acc, c1, c2)          one fresh register pair per instruction (c1, c2 come from the reuse cache)
// form 1: acc = fma2(acc', acc'', acc)     three fresh register pairs
// form 2: acc = fma2(s.F32, acc', acc)     scalar broadcast + two fresh pairs
#include <cstdio>
#include <cuda_runtime.h>
template <int NF2, int NS, int NM, int FORM>
__global__ void __launch_bounds__(128, 3) mix(float *out, int iters, float c)
{
    float2 acc[20];
    float s[4];
    float m[16];
    const float2 c1 = make_float2(c, c * 1.0001f), c2 = make_float2(1e-3f * c, 2e-3f * c);
#pragma unroll
    for (int j = 0; j < 20; ++j) acc[j] = make_float2(threadIdx.x * 1e-3f + j, j * 0.5f);
#pragma unroll
    for (int j = 0; j < 4; ++j) s[j] = threadIdx.x + j;
#pragma unroll
    for (int j = 0; j < 16; ++j) m[j] = 1.5f + threadIdx.x * 1e-3f + j;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int q = 0; q < NF2; ++q) {
            if (FORM == 0) acc[q % 20] = __ffma2_rn(acc[q % 20], c1, c2);              // chain, 1 varying operand
            else if (FORM == 1) acc[q % 20] = __ffma2_rn(acc[(q + 7) % 20], acc[(q + 13) % 20], acc[q % 20]); // 3 distinct reg pairs
            else acc[q % 20] = __ffma2_rn(make_float2(s[q % 4], s[q % 4]), acc[(q + 13) % 20], acc[q % 20]); // scalar broadcast operand
        }
#pragma unroll
        for (int q = 0; q < NS; ++q) s[q % 4] = __fadd_rn(s[q % 4], c);
#pragma unroll
        for (int q = 0; q < NM; ++q) asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(m[q % 16]));
    }
    float r = 0;
#pragma unroll
    for (int j = 0; j < 20; ++j) r += acc[j].x + acc[j].y;
#pragma unroll
    for (int j = 0; j < 4; ++j) r += s[j];
#pragma unroll
    for (int j = 0; j < 16; ++j) r += m[j];
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
}
template <int NF2, int NS, int NM, int FORM> void run(float *out, int ctas_per_sm)
{
    const int iters = 20000;
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    mix<NF2, NS, NM, FORM><<<148 * ctas_per_sm, 128>>>(out, 100, 1.0f);
    cudaEventRecord(a);
    mix<NF2, NS, NM, FORM><<<148 * ctas_per_sm, 128>>>(out, iters, 1.0f);
    cudaEventRecord(b); cudaEventSynchronize(b);
    float ms; cudaEventElapsedTime(&ms, a, b);
    double cyc = ms * 1e-3 * 1.965e9;             // SM cycles
    double per_iter_smsp = cyc / iters;            // cycles per iteration of the warps on one SMSP (ctas_per_sm warps each)
    double fma_cycles = (NF2 * 2 + NS) * ctas_per_sm; // FMA pipe cycles needed per iteration on one SMSP
    double xu_cycles = NM * 8.0 * ctas_per_sm;
    printf("NF2=%2d NS=%d NM=%2d form=%d warps/SMSP=%d : %.1f cyc/iter, FMA need %.0f (%.1f %%), XU need %.0f (%.1f %%)\n", NF2, NS, NM, FORM,
           ctas_per_sm, per_iter_smsp, fma_cycles, 100 * fma_cycles / per_iter_smsp, xu_cycles, 100 * xu_cycles / per_iter_smsp);
}
int main()
{
    float *out; cudaMalloc(&out, 148 * 8 * 128 * 4);
    for (int w = 3; w <= 4; ++w) {
        run<40, 4, 0, 0>(out, w); run<40, 4, 0, 1>(out, w); run<40, 4, 0, 2>(out, w);
        run<40, 4, 2, 1>(out, w); run<40, 4, 4, 1>(out, w); run<40, 4, 6, 1>(out, w); run<40, 4, 8, 1>(out, w);
        run<40, 4, 8, 0>(out, w); run<40, 4, 8, 2>(out, w); run<40, 4, 10, 1>(out, w); run<40, 4, 12, 1>(out, w); run<0, 4, 8, 1>(out, w);
    }
    return 0;
}

// fp32_rate.cu -- FP32 issue-rate (and legacy mma.sync rate) microbenchmark for sm_100a (not part of the library).
//
// Measures how many FP32 lane-operations per clock per SM the FMA pipe sustains for the instruction forms the
// F-engine kernels use (packed FFMA2 / FADD2 / FMUL2, scalar FFMA), with and without operand reuse.
// section 6 derives the "alu" roofline from these numbers; profiles/r1_fp32_rate.txt holds one run.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o fp32_rate fp32_rate.cu   (python -m paper_2303_09886_b200.build --tools)
#include <cstdio>
#include <cuda_runtime.h>
#define ITERS 4096
template <int MODE>
__global__ void k(float *out, float a0, float b0)
{
    // 16 independent accumulators (pairs)
    float2 acc[16];
    float2 s[4];
    float w[8];
    for (int i = 0; i < 16; ++i) acc[i] = make_float2(threadIdx.x * 1e-3f + i, i * 0.5f);
    a0 += threadIdx.x * 1e-6f; b0 += threadIdx.x * 1e-7f;
    for (int i = 0; i < 4; ++i) s[i] = make_float2(a0 + i, a0 - i);
    for (int i = 0; i < 8; ++i) w[i] = b0 + i * 0.01f;
    for (int it = 0; it < ITERS; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            if (MODE == 0) {          // FFMA2 pair * bcast scalar + pair  (FIR form)
                acc[i] = __ffma2_rn(s[i & 3], make_float2(w[i & 7], w[i & 7]), acc[i]);
            } else if (MODE == 1) {   // FFMA2 pair * pair + pair
                acc[i] = __ffma2_rn(s[i & 3], s[(i + 1) & 3], acc[i]);
            } else if (MODE == 2) {   // scalar FFMA x2
                acc[i].x = fmaf(s[i & 3].x, w[i & 7], acc[i].x);
                acc[i].y = fmaf(s[i & 3].y, w[i & 7], acc[i].y);
            } else if (MODE == 3) {   // FADD2
                acc[i] = __fadd2_rn(acc[i], s[i & 3]);
            } else if (MODE == 4) {   // FMUL2 by immediate-like constant
                acc[i] = __fmul2_rn(acc[i], make_float2(1.0000001f, 1.0000001f));
            } else if (MODE == 7) {   // FIR order: one sample pair against 16 weights: ptxas marks the sample .reuse
                acc[i] = __ffma2_rn(s[0], make_float2(w[i & 7] , w[i & 7]), acc[i]);
            } else if (MODE == 5) {   // FFMA2 acc = acc*s + acc (2 distinct pairs)
                acc[i] = __ffma2_rn(acc[i], s[i & 3], acc[i]);
            }
        }
    }
    float r = 0;
    for (int i = 0; i < 16; ++i) r += acc[i].x + acc[i].y;
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
}
template <int MODE>
void run(const char *name, int threads, int ctas_per_sm)
{
    float *out;
    cudaMalloc(&out, 148 * 32 * 1024 * sizeof(float));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    int grid = 148 * ctas_per_sm;
    k<MODE><<<grid, threads>>>(out, 1.0f, 0.5f);
    cudaDeviceSynchronize();
    cudaEventRecord(e0);
    for (int r = 0; r < 5; ++r) k<MODE><<<grid, threads>>>(out, 1.0f, 0.5f);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1); ms /= 5;
    double lane_ops = (double)grid * threads * ITERS * 16 * 2;     // lane-FMAs (or adds)
    double per_clk_sm = lane_ops / (ms * 1e-3) / 148 / 1.965e9;
    printf("%-28s threads=%4d ctas/sm=%d  %.3f ms  %.1f lane-ops/clk/SM (at 1.965 GHz)  %.2f T lane-ops/s\n", name, threads, ctas_per_sm, ms, per_clk_sm, lane_ops / (ms * 1e-3) / 1e12);
    cudaFree(out);
}
// legacy tensor path: mma.sync.m16n8k16 f16 x f16 + f32 (what a tensor-core FIR would use)
__global__ void k_hmma(float *out, unsigned a0)
{
    unsigned a[4] = {a0 + threadIdx.x, a0 ^ 0x3c003c00u, a0 + 7, a0 + 9};
    unsigned b[2] = {0x3c003c00u, 0x38003800u};
    float d[8][4];
    for (int i = 0; i < 8; ++i) for (int j = 0; j < 4; ++j) d[i][j] = 0.f;
    for (int it = 0; it < ITERS; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                         : "+f"(d[i][0]), "+f"(d[i][1]), "+f"(d[i][2]), "+f"(d[i][3])
                         : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
    }
    float r = 0;
    for (int i = 0; i < 8; ++i) for (int j = 0; j < 4; ++j) r += d[i][j];
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
}
int main()
{
    for (int t : {128, 256, 512, 1024}) {
        run<0>("FFMA2 pair*bcast+pair", t, 1);
        run<1>("FFMA2 pair*pair+pair", t, 1);
        run<2>("FFMA scalar x2", t, 1);
        run<3>("FADD2", t, 1);
        run<4>("FMUL2 const", t, 1);
        run<5>("FFMA2 acc*s+acc", t, 1);
        run<7>("FFMA2 s0*bcast+pair (reuse)", t, 1);
    }
    {
        float *out;
        cudaMalloc(&out, 148 * 1024 * 4 * sizeof(float));
        for (int threads : {128, 256, 512, 1024}) {
            cudaEvent_t e0, e1;
            cudaEventCreate(&e0); cudaEventCreate(&e1);
            k_hmma<<<148, threads>>>(out, 0x3c00u);
            cudaDeviceSynchronize();
            cudaEventRecord(e0);
            for (int r = 0; r < 5; ++r) k_hmma<<<148, threads>>>(out, 0x3c00u);
            cudaEventRecord(e1);
            cudaEventSynchronize(e1);
            float ms; cudaEventElapsedTime(&ms, e0, e1); ms /= 5;
            const double mmas = 148.0 * (threads / 32) * ITERS * 8;
            printf("mma.sync m16n8k16 f16        threads=%4d ctas/sm=1  %.3f ms  %.1f TFLOP/s  %.2f cycles per HMMA per SMSP (at 1.965 GHz)\n",
                   threads, ms, mmas * 2.0 * 16 * 8 * 16 / (ms * 1e-3) / 1e12, (ms * 1e-3 * 1.965e9) / (ITERS * 8.0 * (threads / 32) / 4.0));
        }
        cudaFree(out);
    }
    return 0;
}

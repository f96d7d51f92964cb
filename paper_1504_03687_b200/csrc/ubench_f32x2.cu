// ubench_f32x2.cu -- issue cost of the packed FP32 instructions of the force kernel by operand pattern.
//
// Evidence for DESIGN.md section 7 ("what bounds the pair loop"): the force kernel's 27 (local frame) or
// 33 (hi/lo) packed instructions per (2 i x 1 j) do not all cost the 2 pipe cycles of an FFMA2: an
// instruction that reads three DISTINCT register pairs waits for the register file.  This standalone
// program (not part of libnbreg) times independent chains of one instruction form per kernel:
//
//     nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o /tmp/ubench_f32x2 \
//          paper_1504_03687_b200/csrc/ubench_f32x2.cu && /tmp/ubench_f32x2
//     cuobjdump -sass /tmp/ubench_f32x2 | grep -E "FFMA2|FADD2|FMUL2|FFMA " | sort | uniq -c | sort -rn | head
//
// Output: cycles per instruction and warp scheduler (SMSP) with 1, 2 and 4 warps per SMSP; the 4-warp
// column is the throughput figure.  Summary of a B200 run: profiles/r02_ubench_f32x2.md.
#include <cstdio>
#include <cuda_runtime.h>

enum Form {
    FFMA2_3PAIRS = 0,   // c = a * b + c, three distinct register pairs                (acc, jerk, r.v chains)
    FFMA2_SHARED,       // one pair shared by consecutive instructions (operand reuse cache)
    FFMA2_2PAIRS,       // c = a * a + c                                               (r^2 chain)
    FFMA_SCALAR_X2,     // the same work as two scalar FFMA
    FFMA2_BCAST,        // one operand a 32-bit scalar broadcast to both halves (SASS R.F32: the j side)
    FADD2_2PAIRS,       // c = a + c                                                   (differences)
    FMUL2_2PAIRS,       // c = a * c
    NFORMS
};

template <int FORM>
__global__ void chains(float2 *out, int iters, float s, long long *cycles) {
    float2 a[8], b[8], c[8];
    for (int i = 0; i < 8; ++i) {
        a[i] = make_float2(threadIdx.x * 1e-3f + i, s + i);
        b[i] = make_float2(s * i + 1.f + threadIdx.x * 1e-4f, 0.5f + i * s + threadIdx.x * 1e-5f);
        c[i] = make_float2(0.f, 1.f);
    }
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {      // eight independent chains: latency is hidden, issue is measured
            if (FORM == FFMA2_3PAIRS) c[i] = __ffma2_rn(a[i], b[i], c[i]);
            if (FORM == FFMA2_SHARED) c[i] = __ffma2_rn(a[0], b[i], c[i]);
            if (FORM == FFMA2_2PAIRS) c[i] = __ffma2_rn(a[i], a[i], c[i]);
            if (FORM == FFMA_SCALAR_X2) {
                c[i].x = __fmaf_rn(a[i].x, b[i].x, c[i].x);
                c[i].y = __fmaf_rn(a[i].y, b[i].y, c[i].y);
            }
            if (FORM == FFMA2_BCAST) c[i] = __ffma2_rn(a[i], make_float2(b[i].x, b[i].x), c[i]);
            if (FORM == FADD2_2PAIRS) c[i] = __fadd2_rn(a[i], c[i]);
            if (FORM == FMUL2_2PAIRS) c[i] = __fmul2_rn(a[i], c[i]);
        }
    }
    const long long t1 = clock64();
    float2 r = make_float2(0, 0);
    for (int i = 0; i < 8; ++i) { r.x += c[i].x; r.y += c[i].y; }
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
    if (threadIdx.x == 0 && blockIdx.x == 0) *cycles = t1 - t0;
}

template <int FORM>
double run(float2 *out, long long *d_cycles, int warps_per_smsp, int sms) {
    const int iters = 4096;
    long long h = 0;
    chains<FORM><<<sms, 128 * warps_per_smsp>>>(out, iters, 0.25f, d_cycles);      // warm-up
    chains<FORM><<<sms, 128 * warps_per_smsp>>>(out, iters, 0.25f, d_cycles);
    cudaMemcpy(&h, d_cycles, sizeof(h), cudaMemcpyDeviceToHost);
    return (double)h / (iters * 8.0) / warps_per_smsp;      // cycles per instruction per SMSP
}

int main() {
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, 0) != cudaSuccess) { printf("no CUDA device\n"); return 1; }
    float2 *out;
    long long *d_cycles;
    cudaMalloc(&out, sizeof(float2) * 512 * prop.multiProcessorCount);
    cudaMalloc(&d_cycles, sizeof(long long));
    const char *name[NFORMS] = {"FFMA2  3 distinct pairs", "FFMA2  1 pair shared (reuse)", "FFMA2  2 distinct pairs",
                                "2 x FFMA (scalar)", "FFMA2  scalar-broadcast operand", "FADD2  2 pairs", "FMUL2  2 pairs"};
    printf("%s, %d SMs, cycles per instruction per SMSP\n", prop.name, prop.multiProcessorCount);
    printf("%-34s %10s %10s %10s\n", "form", "1 warp", "2 warps", "4 warps");
    for (int f = 0; f < NFORMS; ++f) {
        double r[3];
        int k = 0;
        for (int w = 1; w <= 4; w *= 2) {
            const int sms = prop.multiProcessorCount;
            switch (f) {
                case 0: r[k] = run<0>(out, d_cycles, w, sms); break;
                case 1: r[k] = run<1>(out, d_cycles, w, sms); break;
                case 2: r[k] = run<2>(out, d_cycles, w, sms); break;
                case 3: r[k] = run<3>(out, d_cycles, w, sms); break;
                case 4: r[k] = run<4>(out, d_cycles, w, sms); break;
                case 5: r[k] = run<5>(out, d_cycles, w, sms); break;
                default: r[k] = run<6>(out, d_cycles, w, sms); break;
            }
            ++k;
        }
        printf("%-34s %10.3f %10.3f %10.3f\n", name[f], r[0], r[1], r[2]);
    }
    return cudaDeviceSynchronize() == cudaSuccess ? 0 : 1;
}

// pipe_probe.cu -- stand-alone probe of the sm_100a pipes that bound the RBE k-space kernels
// (SURVEY.md s7 stage 6: the roofline needs the FP32-FMA, IMAD and MUFU issue peaks, which
// MEASURED_PEAKS.json does not hold), and of the accuracy of MUFU.SIN / MUFU.COS on the exact
// phase pipeline the kernels use (32-bit fixed-point turns -> I2FP -> FMUL -> sin/cos.approx).
//
//   build:  python -m paper_2407_09315_b200.build   (-> paper_2407_09315_b200/pipe_probe)
//   run:    ./paper_2407_09315_b200/pipe_probe > profiles/<round>_pipe_probe.txt   (on a B200)
//
// Part 1 prints SM-sub-partition cycles per warp instruction for dependent-free chains
// (8 independent chains per thread, 8 warps per sub-partition), assuming the max SM clock.
// Part 2 prints the error statistics of cos/sin over a full turn (2^22 phases), in particular
// the MEAN error of MUFU.COS: it is what forces the structure-factor kernel to alternate the
// sign of its pair amplitudes (rbe_kernels.cuh, "half a turn on every other pair").
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <vector>
#include <cuda_runtime.h>

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { printf("CUDA error %s at line %d\n", cudaGetErrorString(e_), __LINE__); exit(1); } } while (0)

__device__ __forceinline__ float mufu_sin(float x) { float r; asm volatile("sin.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float mufu_cos(float x) { float r; asm volatile("cos.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float mufu_ex2(float x) { float r; asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

enum Mode { FFMA = 0, IMAD = 1, FFMA_IMAD = 2, EX2 = 3, FFMA_EX2 = 4, SIN = 5, I2FP = 6, IMAD_EX2 = 7 };

// C independent chains per thread; per chain and iteration: NF ops of the mode (+1 MUFU for the mixes)
template <int MODE, int C, int NF>
__global__ void __launch_bounds__(256) rate_kernel(float* out, int iters, float a, float b, int ia, int ib) {
    float v[C]; int w[C];
#pragma unroll
    for (int c = 0; c < C; ++c) { v[c] = threadIdx.x * 0.001f + c; w[c] = threadIdx.x + c; }
    const float bb[4] = {b, b + 1.f, b + 2.f, b + 3.f};
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int c = 0; c < C; ++c) {
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                if (MODE == FFMA || MODE == FFMA_EX2) v[c] = fmaf(v[c], a, bb[f & 3]);
                if (MODE == IMAD || MODE == IMAD_EX2) w[c] = w[c] * ia + ib;
                if (MODE == FFMA_IMAD) { v[c] = fmaf(v[c], a, bb[f & 3]); w[c] = w[c] * ia + ib; }
                if (MODE == I2FP) w[c] = __float_as_int((float)w[c]);
            }
            if (MODE == EX2 || MODE == FFMA_EX2) v[c] = mufu_ex2(v[c]);
            if (MODE == IMAD_EX2) { v[c] = mufu_ex2(v[c]); w[c] ^= __float_as_int(v[c]); }
            if (MODE == SIN) v[c] = mufu_sin(v[c]);
        }
    }
    float s = 0.f; int t = 0;
#pragma unroll
    for (int c = 0; c < C; ++c) { s += v[c]; t += w[c]; }
    out[blockIdx.x * blockDim.x + threadIdx.x] = s + t;
}

static int g_sms = 148;
static double g_clk = 1.965e9;

template <int MODE, int C, int NF>
static void rate(const char* name, int instr_per_chain_iter, float* d_out) {
    const int iters = 4096, threads = 256, ctas_per_sm = 4;   // 8 warps per sub-partition
    auto launch = [&]() { rate_kernel<MODE, C, NF><<<g_sms * ctas_per_sm, threads>>>(d_out, iters, 1.0001f, 0.5f, 3, 7); };
    cudaEvent_t e0, e1; CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    launch(); CK(cudaDeviceSynchronize());
    CK(cudaEventRecord(e0)); launch(); launch(); launch(); CK(cudaEventRecord(e1)); CK(cudaDeviceSynchronize());
    float ms; CK(cudaEventElapsedTime(&ms, e0, e1)); ms /= 3;
    const double warp_chain_iters = (double)g_sms * ctas_per_sm * threads / 32 * C * iters;
    const double cyc = ms * 1e-3 * g_clk * g_sms * 4 / warp_chain_iters;
    printf("%-28s %7.2f cycles per chain-iteration (%2d instr): %5.2f cycles/instr per sub-partition -> %6.1f lanes/SM/clk\n",
           name, cyc, instr_per_chain_iter, cyc / instr_per_chain_iter, 128.0 * instr_per_chain_iter / cyc);
}

__global__ void sincos_kernel(float2* out, int n, uint32_t stride, uint32_t base) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    // the kernels' phase pipeline: int32 turns -> I2FP -> FMUL(K) -> [FMUL.RZ(1/2pi) -> MUFU]
    const float K = (float)(1.0 / (4294967296.0 * 0.15915493667125701904));
    const uint32_t ph = base + (uint32_t)i * stride;
    const float x = (float)(int32_t)ph * K;
    out[i] = make_float2(mufu_cos(x), mufu_sin(x));
}

int main() {
    cudaDeviceProp prop; CK(cudaGetDeviceProperties(&prop, 0));
    g_sms = prop.multiProcessorCount;
    int khz = 0; CK(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0));
    g_clk = khz * 1e3;
    printf("# pipe_probe: %s, %d SMs, max SM clock %.0f MHz (cycle counts assume it)\n", prop.name, g_sms, khz / 1e3);
    float* d_out; CK(cudaMalloc(&d_out, (size_t)64 << 20));

    printf("## part 1: issue rates\n");
    rate<FFMA, 8, 8>("FFMA", 8, d_out);
    rate<IMAD, 8, 8>("IMAD", 8, d_out);
    rate<I2FP, 8, 8>("I2FP.F32.S32", 8, d_out);
    rate<FFMA_IMAD, 8, 4>("FFMA + IMAD, 1:1", 8, d_out);
    rate<EX2, 8, 1>("MUFU.EX2", 1, d_out);
    rate<SIN, 8, 1>("FMUL.RZ + MUFU.SIN", 2, d_out);
    rate<FFMA_EX2, 8, 4>("4 FFMA + MUFU", 5, d_out);
    rate<FFMA_EX2, 8, 8>("8 FFMA + MUFU", 9, d_out);
    rate<FFMA_EX2, 8, 16>("16 FFMA + MUFU", 17, d_out);
    rate<FFMA_EX2, 8, 24>("24 FFMA + MUFU", 25, d_out);
    rate<IMAD_EX2, 8, 6>("6 IMAD + MUFU + LOP", 8, d_out);

    printf("## part 2: MUFU.COS / MUFU.SIN error over one turn (phase pipeline of the kernels)\n");
    const int n = 1 << 22;
    float2* d_sc; CK(cudaMalloc(&d_sc, (size_t)n * sizeof(float2)));
    std::vector<float2> h(n);
    for (int pass = 0; pass < 2; ++pass) {
        const uint32_t base = pass ? 0x167u : 0u;   // pass 1: phases that are not exactly representable in fp32
        sincos_kernel<<<n / 256, 256>>>(d_sc, n, 1u << 10, base);
        CK(cudaMemcpy(h.data(), d_sc, (size_t)n * sizeof(float2), cudaMemcpyDeviceToHost));
        double mc = 0, ms = 0, rc = 0, rs = 0, xc = 0, xs = 0, rad = 0;
        for (int i = 0; i < n; ++i) {
            const uint32_t ph = base + (uint32_t)i * 1024u;
            const double t = (double)(int32_t)ph / 4294967296.0 * 6.283185307179586476925287;
            const double ec = (double)h[i].x - cos(t), es = (double)h[i].y - sin(t);
            mc += ec; ms += es; rc += ec * ec; rs += es * es;
            xc = fmax(xc, fabs(ec)); xs = fmax(xs, fabs(es));
            rad += ec * cos(t) + es * sin(t);
        }
        printf("pass %d: cos error mean %+.3e rms %.3e max %.3e | sin error mean %+.3e rms %.3e max %.3e | radial mean %+.3e\n",
               pass, mc / n, sqrt(rc / n), xc, ms / n, sqrt(rs / n), xs, rad / n);
    }
    return 0;
}

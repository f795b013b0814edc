// hot_peak.cu -- the roofline denominator of the interaction kernels, measured on the device in use:
// a register-only chain of fused multiply-adds (scalar FFMA and packed FFMA2), 8 independent chains
// per thread, 16 warps per SM.  bench.py reports it beside the peak derived from unit counts and the
// clock (148 SMs x 128 lanes x 2 flops x clocks.max.sm) -- DESIGN.md "Roofline".
#include "hot_internal.h"

template <bool PACKED>
__global__ void __launch_bounds__(128) fma_chain_kernel(float* __restrict__ out, int iters, float b, float c) {
    float s = 0.f;
    if (PACKED) {
        unsigned long long a[8], bb, cc;
        asm("mov.b64 %0, {%1, %1};" : "=l"(bb) : "f"(b));
        asm("mov.b64 %0, {%1, %1};" : "=l"(cc) : "f"(c));
#pragma unroll
        for (int k = 0; k < 8; ++k) asm("mov.b64 %0, {%1, %2};" : "=l"(a[k]) : "f"(threadIdx.x * 1e-3f + k), "f"(1.0f + k));
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int k = 0; k < 8; ++k) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(a[k]) : "l"(bb), "l"(cc));
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) { float x, y; asm("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(a[k])); s += x + y; }
    } else {
        float a[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) a[k] = threadIdx.x * 1e-3f + k;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int k = 0; k < 8; ++k) a[k] = fmaf(a[k], b, c);
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) s += a[k];
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// The same pipe with operands that come from the register file: the packed instructions read their register operands at
// 64 bits per lane and clock, so one with three different 64-bit register sources occupies the pipe for three clocks
// instead of two (a scalar FFMA with three different sources: 1.5 instead of 1).  MODE 0: d = a_k * a_k + d (two reads),
// 1: d = a_k * b_k + d (three reads), 2: scalar d = a_k * b_k + d.  This is what bounds the interaction kernels'
// inner loops below the FMA peak.
template <int MODE>
__global__ void __launch_bounds__(128) fma_operand_kernel(float* __restrict__ out, const float* __restrict__ in, int iters) {
    float s = 0.f;
    const float* p = in + threadIdx.x * 48;
    if (MODE < 2) {
        unsigned long long a[8], b[8], d[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            asm volatile("mov.b64 %0, {%1, %2};" : "=l"(a[k]) : "f"(p[2 * k]), "f"(p[2 * k + 1]));
            asm volatile("mov.b64 %0, {%1, %2};" : "=l"(b[k]) : "f"(p[16 + 2 * k]), "f"(p[17 + 2 * k]));
            asm volatile("mov.b64 %0, {%1, %2};" : "=l"(d[k]) : "f"(p[32 + 2 * k]), "f"(p[33 + 2 * k]));
        }
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    if (MODE == 0) asm volatile("fma.rn.f32x2 %0, %1, %1, %0;" : "+l"(d[k]) : "l"(a[k]));
                    else asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(d[k]) : "l"(a[k]), "l"(b[k]));
                }
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) { float x, y; asm("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(d[k])); s += x + y; }
    } else {
        float a[16], b[16], d[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) { a[k] = p[k]; b[k] = p[16 + k]; d[k] = p[32 + k]; }
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int k = 0; k < 16; ++k) asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(d[k]) : "f"(a[k]), "f"(b[k]));
        }
#pragma unroll
        for (int k = 0; k < 16; ++k) s += d[k];
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}
cudaError_t measure_fp32_operands(double* tf3, cudaStream_t st) { // tf3[0..2]: TFLOP/s of MODE 0, 1, 2 (FMA = 2 flops)
    int dev = 0, nsm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    const int blocks = nsm * 4, iters = 2048;
    float *out = nullptr, *in = nullptr;
    cudaError_t e = cudaMalloc(&out, sizeof(float) * (size_t)blocks * 128);
    if (e != cudaSuccess) return e;
    e = cudaMalloc(&in, sizeof(float) * 128 * 48);
    if (e != cudaSuccess) { cudaFree(out); return e; }
    {
        float h[128 * 48];
        for (int i = 0; i < 128 * 48; ++i) h[i] = 1.0f + 1e-6f * (float)(i % 977);
        cudaMemcpyAsync(in, h, sizeof(h), cudaMemcpyHostToDevice, st);
        cudaStreamSynchronize(st);
    }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    for (int mode = 0; mode < 3 && e == cudaSuccess; ++mode)
        for (int rep = 0; rep < 2; ++rep) { // the first run warms up
            cudaEventRecord(e0, st);
            if (mode == 0) fma_operand_kernel<0><<<blocks, 128, 0, st>>>(out, in, iters);
            else if (mode == 1) fma_operand_kernel<1><<<blocks, 128, 0, st>>>(out, in, iters);
            else fma_operand_kernel<2><<<blocks, 128, 0, st>>>(out, in, iters);
            cudaEventRecord(e1, st);
            e = cudaEventSynchronize(e1);
            if (e != cudaSuccess) break;
            float ms = 0;
            cudaEventElapsedTime(&ms, e0, e1);
            tf3[mode] = (double)blocks * 128 * iters * 64 * (mode < 2 ? 2 : 1) * 2 / (ms * 1e-3) / 1e12;
        }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out); cudaFree(in);
    if (e == cudaSuccess) e = cudaGetLastError();
    return e;
}

// TFLOP/s of the two chains (FMA = 2 flops), timed with CUDA events on `st`; ~10 ms of device time
cudaError_t measure_fp32(double* tf_scalar, double* tf_packed, cudaStream_t st) {
    int dev = 0, nsm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    const int blocks = nsm * 4, iters = 4096;
    float* out = nullptr;
    cudaError_t e = cudaMalloc(&out, sizeof(float) * (size_t)blocks * 128);
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double res[2] = {0, 0};
    for (int packed = 0; packed < 2; ++packed) {
        for (int rep = 0; rep < 2; ++rep) { // the first run warms up
            cudaEventRecord(e0, st);
            if (packed) fma_chain_kernel<true><<<blocks, 128, 0, st>>>(out, iters, 1.0001f, 1e-9f);
            else fma_chain_kernel<false><<<blocks, 128, 0, st>>>(out, iters, 1.0001f, 1e-9f);
            cudaEventRecord(e1, st);
            e = cudaEventSynchronize(e1);
            if (e != cudaSuccess) break;
            float ms = 0;
            cudaEventElapsedTime(&ms, e0, e1);
            res[packed] = (double)blocks * 128 * iters * 64 * (packed ? 2 : 1) * 2 / (ms * 1e-3) / 1e12;
        }
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    if (e == cudaSuccess) e = cudaGetLastError();
    *tf_scalar = res[0]; *tf_packed = res[1];
    return e;
}

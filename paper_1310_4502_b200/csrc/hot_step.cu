// hot_step.cu -- f-4: the "kick" and "drift" operators around the force call (symplectic integration in a
// comoving background; the two time factors -- integrals over the expansion history there -- are the caller's).
//   v <- v + a dtk,   x <- x + v dtd,   one fused multiply-add each in fp32; periodic boxes wrap x into [lo, lo + size).
// Streaming, HBM-bound: 36 B read + 24 B written per body, 128-bit accesses.
#include "hot_internal.h"

__device__ __forceinline__ float wrap_coord(float x, float l, float size) {
    const float t = __fsub_rn(x, l);
    const float q = floorf(__fdiv_rn(t, size));
    x = __fadd_rn(fmaf(-q, size, t), l);
    if (x >= __fadd_rn(l, size)) x = l; // rounding may land on the upper face
    if (x < l) x = l;
    return x;
}
__global__ void __launch_bounds__(256) kick_drift_kernel(float* __restrict__ pos, float* __restrict__ vel, const float* __restrict__ acc,
                                                         int64_t n3, float dtk, float dtd, float lox, float loy, float loz, float size,
                                                         int periodic, int vec) {
    const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; // 4 consecutive floats of the [n][3] arrays
    const int64_t i0 = 4 * q;
    if (i0 >= n3) return;
    float p[4], v[4], a[4];
    const int cnt = (int)min((int64_t)4, n3 - i0);
    if (vec && cnt == 4) {
        const float4 P4 = reinterpret_cast<const float4*>(pos)[q], V4 = reinterpret_cast<const float4*>(vel)[q], A4 = __ldg(reinterpret_cast<const float4*>(acc) + q);
        p[0] = P4.x; p[1] = P4.y; p[2] = P4.z; p[3] = P4.w; v[0] = V4.x; v[1] = V4.y; v[2] = V4.z; v[3] = V4.w;
        a[0] = A4.x; a[1] = A4.y; a[2] = A4.z; a[3] = A4.w;
    } else {
        for (int k = 0; k < cnt; ++k) { p[k] = pos[i0 + k]; v[k] = vel[i0 + k]; a[k] = acc[i0 + k]; }
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        if (k < cnt) {
            v[k] = fmaf(a[k], dtk, v[k]);
            p[k] = fmaf(v[k], dtd, p[k]);
            if (periodic) { const int ax = (int)((i0 + k) % 3); p[k] = wrap_coord(p[k], ax == 0 ? lox : ax == 1 ? loy : loz, size); }
        }
    }
    if (vec && cnt == 4) {
        reinterpret_cast<float4*>(pos)[q] = make_float4(p[0], p[1], p[2], p[3]);
        reinterpret_cast<float4*>(vel)[q] = make_float4(v[0], v[1], v[2], v[3]);
    } else {
        for (int k = 0; k < cnt; ++k) { pos[i0 + k] = p[k]; vel[i0 + k] = v[k]; }
    }
}
cudaError_t launch_kick_drift(float* pos, float* vel, const float* acc, int64_t n, float dtk, float dtd, float lox, float loy, float loz,
                              float size, int periodic, cudaStream_t st) {
    const int64_t n3 = 3 * n, quads = (n3 + 3) / 4;
    const int vec = ((reinterpret_cast<uintptr_t>(pos) | reinterpret_cast<uintptr_t>(vel) | reinterpret_cast<uintptr_t>(acc)) & 15u) == 0;
    HOT_LAUNCHED(1);
    kick_drift_kernel<<<(unsigned)((quads + 255) / 256), 256, 0, st>>>(pos, vel, acc, n3, dtk, dtd, lox, loy, loz, size, periodic, vec);
    return cudaGetLastError();
}

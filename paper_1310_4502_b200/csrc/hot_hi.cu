// hot_hi.cu -- f-3: expansion orders p = 6 and 8 ("interaction routines through p=8 without human
// intervention", :267 Fig 6).  Orders 0-4 of every accepted cell are evaluated by hot_forces.cu; this kernel ADDS the
// terms of degree 5 .. P, whose code (hi_terms<P>) and per-cell record (hi_record<P>, built by the upward pass) come from
// the generator gen_hi_orders.py.  One warp per sink group, up to 8 sinks per lane, one cell at a time: its record
// (84 / 249 floats) is staged in shared memory and read as broadcasts by the generated straight-line code.
// Not a bandwidth or pipe-tuned kernel: ~500 / ~1900 flops per interaction, the high orders are an accuracy feature.
#include "hot_internal.h"
#define HOT_HI_WITH_TERMS
#include "hot_hi_generated.inc"

#define HI_WARPS 4
#define HI_SINKS 8 // per lane: 256 = HOT_MAX_NCRIT sinks per pass

int hi_record_floats(int order) { return order >= 8 ? HiOrder<8>::NT : HiOrder<6>::NT; }
int hi_raw_floats(int order) { return order >= 8 ? HiOrder<8>::NRAW : HiOrder<6>::NRAW; }

template <int P, bool PER>
__global__ void __launch_bounds__(HI_WARPS * 32) forces_hi_kernel(const __grid_constant__ ForceArgs A, const float* __restrict__ hiT, int stride) {
    constexpr int NT = HiOrder<P>::NT;
    __shared__ float s_T[HI_WARPS][NT + 8];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    float* const T = s_T[w];
    for (int64_t gi = A.g0 + (int64_t)blockIdx.x * HI_WARPS + w; gi < A.g1; gi += (int64_t)gridDim.x * HI_WARPS) {
        const GroupRec g = A.group[gi];
        // origin of the relative coordinates: the centre of the group cube (as in hot_forces.cu)
        double ox, oy, oz;
        {
            const WalkCell gw = A.wcell[g.cell];
            const int gs = 1 << (HOT_MAXLEVEL - (int)(gw.w >> 27));
            const int gox = (int)(gw.x & 0x1fffffu), goy = (int)((gw.x >> 21) | ((gw.y & 0x3ffu) << 11)), goz = (int)((gw.y >> 10) & 0x1fffffu);
            const double h = A.size * (1.0 / 2097152.0);
            ox = A.lo[0] + ((double)gox + 0.5 * gs) * h; oy = A.lo[1] + ((double)goy + 0.5 * gs) * h; oz = A.lo[2] + ((double)goz + 0.5 * gs) * h;
        }
        const unsigned long long o0 = A.pcoff[gi];
        const int n = (int)A.lpc[gi];
        for (uint32_t s0 = 0; s0 < g.count; s0 += 32 * HI_SINKS) { // finest-level groups can exceed 256 bodies
            float x[HI_SINKS][3], a[HI_SINKS][4];
#pragma unroll
            for (int i = 0; i < HI_SINKS; ++i) {
                const uint32_t loc = s0 + 32 * i + lane;
                const float4 b = A.body[g.first + (loc < g.count ? loc : 0u)];
                x[i][0] = (float)((double)b.x - ox); x[i][1] = (float)((double)b.y - oy); x[i][2] = (float)((double)b.z - oz);
                a[i][0] = a[i][1] = a[i][2] = a[i][3] = 0.0f;
            }
            const int ns = (int)min((uint32_t)HI_SINKS, (g.count - s0 + 31u) / 32u); // sink slots in use (warp-uniform)
            for (int j = 0; j < n; ++j) {
                const uint32_t c = A.pclist[o0 + j] & 0x0fffffffu;
                __syncwarp();
                for (int q = lane; q < NT; q += 32) T[q] = hiT[(size_t)c * stride + q];
                if (lane == 0) {
                    const CellA cA = A.cellA[c];
                    double shx = 0, shy = 0, shz = 0;
                    if (PER) { const int im = A.pcimg[o0 + j]; shx = (double)(im / 25 - 2) * A.size; shy = (double)((im / 5) % 5 - 2) * A.size; shz = (double)(im % 5 - 2) * A.size; }
                    T[NT] = (float)(ox - (cA.zx + shx)); T[NT + 1] = (float)(oy - (cA.zy + shy)); T[NT + 2] = (float)(oz - (cA.zz + shz));
                    T[NT + 3] = (float)ldexp(A.size, -(int)(A.wcell[c].w >> 27)); // the cell's side
                }
                __syncwarp();
                const float nzx = T[NT], nzy = T[NT + 1], nzz = T[NT + 2], side = T[NT + 3];
#pragma unroll 1
                for (int i = 0; i < ns; ++i) {
                    const float Rx = x[i][0] + nzx, Ry = x[i][1] + nzy, Rz = x[i][2] + nzz;
                    const float ri = rsqrtf(fmaf(Rx, Rx, fmaf(Ry, Ry, fmaf(Rz, Rz, A.spline ? 0.0f : A.eps2))));
                    hi_terms<P>(T, Rx * ri, Ry * ri, Rz * ri, ri, side * ri, a[i][0], a[i][1], a[i][2], a[i][3]);
                }
            }
#pragma unroll
            for (int i = 0; i < HI_SINKS; ++i) {
                const uint32_t loc = s0 + 32 * i + lane;
                if (loc < g.count) {
                    const uint32_t o = A.perm[g.first + loc];
                    A.acc[3 * (int64_t)o] += a[i][0]; A.acc[3 * (int64_t)o + 1] += a[i][1]; A.acc[3 * (int64_t)o + 2] += a[i][2];
                    if (A.pot) A.pot[o] += a[i][3];
                }
            }
        }
    }
}

cudaError_t launch_forces_hi(const ForceArgs& a, int P, const float* hiT, int hi_stride, cudaStream_t st) {
    const int64_t ng = a.g1 - a.g0;
    if (ng <= 0) return cudaSuccess;
    int64_t nb = (ng + HI_WARPS - 1) / HI_WARPS;
    if (nb > 148 * 32) nb = 148 * 32;
    HOT_LAUNCHED(1);
    if (P >= 8) {
        if (a.periodic) forces_hi_kernel<8, true><<<(unsigned)nb, HI_WARPS * 32, 0, st>>>(a, hiT, hi_stride);
        else forces_hi_kernel<8, false><<<(unsigned)nb, HI_WARPS * 32, 0, st>>>(a, hiT, hi_stride);
    } else {
        if (a.periodic) forces_hi_kernel<6, true><<<(unsigned)nb, HI_WARPS * 32, 0, st>>>(a, hiT, hi_stride);
        else forces_hi_kernel<6, false><<<(unsigned)nb, HI_WARPS * 32, 0, st>>>(a, hiT, hi_stride);
    }
    return cudaGetLastError();
}

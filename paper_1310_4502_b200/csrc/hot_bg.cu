// hot_bg.cu -- f-1: per-cell background subtraction for periodic boxes (Fig 2; R-18).
//
//   bg_moments_kernel : per cell, the moments about the cell CENTRE (parallel-axis shift of the centre-of-mass moments of
//                       the upward pass) minus those of the uniform cube of the mean density, through the same order
//                       (PAPER.md:86); the dipole is present.  fp64 arithmetic, fp32 records.
//   forces_bg_kernel  : per sink, in fp64: the far field of hot_periodic.cu + the background added back in closed form,
//                       rhobar x [homogeneous (5 L)^3 cube - homogeneous near cube K_G] ("removed analytically", Fig 2;
//                       refs [59, 46]) + the virtual cubes (empty octants, cubes of rejected leaves: only the negative
//                       background; few) -> farc[].  The flagged cells of the walk (most of a periodic run's
//                       interactions) are evaluated about their centres, with the dipole, by the blocked kernel of
//                       hot_forces.cu (its BGV variant), which adds its fp64 sums to farc[]; the launch over the plain near
//                       field then adds farc[] to its own fp64 sums before the one rounding to fp32.
//                       (with_cells = 1 makes this kernel evaluate the flagged cells too: the plain form the blocked one was
//                       checked against, 2.4 x slower.)
// One warp per sink group, sinks one per lane, entries one at a time through shared memory.
#include "hot_interact.cuh"

__host__ __device__ constexpr int bidx(int a, int b, int c) {
    int d = a + b + c;
    return d * (d + 1) * (d + 2) / 6 + (d - a) * (d - a + 1) / 2 + (d - a - b);
}
__device__ __forceinline__ double cube1d(int a, double s) { // int_{-s/2}^{s/2} x^a dx
    if (a & 1) return 0.0;
    double h = 0.5 * s, p = h;
    for (int k = 0; k < a; ++k) p *= h;
    return 2.0 * p / (double)(a + 1);
}
// record of a background-subtracted cell as the scalar pc_one stages it: q0 = (-cx, -cy, -cz, -dM0) is formed by the caller
struct BgRec { float m0, d1x, d1y, d1z; CellM2 E2; CellM34 M34; };

template <int ORDER>
__global__ void __launch_bounds__(128) bg_moments_kernel(const WalkCell* __restrict__ wcell, const CellA* __restrict__ cellA, const double* __restrict__ m0d,
                                                         const CellM2* __restrict__ cellM2, const CellM34* __restrict__ cellM34,
                                                         int64_t ncells, double lox, double loy, double loz, double size, double rhobar,
                                                         float4* __restrict__ bgA, CellM2* __restrict__ bgE2, CellM34* __restrict__ bgM34) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncells) return;
    const WalkCell wc = wcell[c];
    const int lev = (int)(wc.w >> 27);
    const double h = size * (1.0 / 2097152.0), side = ldexp(size, -lev);
    const double cx = lox + (double)(wc.x & 0x1fffffu) * h + 0.5 * side;
    const double cy = loy + (double)((wc.x >> 21) | ((wc.y & 0x3ffu) << 11)) * h + 0.5 * side;
    const double cz = loz + (double)((wc.y >> 10) & 0x1fffffu) * h + 0.5 * side;
    const CellA A = cellA[c];
    const double m0 = m0d[c], dx = A.zx - cx, // the fp64 mass: mass - rhobar s^3 is a small difference for the coarse cells
                  dy = A.zy - cy, dz = A.zz - cz; // centre of mass relative to the cell centre
    constexpr int P = ORDER >= 4 ? 4 : (ORDER >= 2 ? 2 : 1);
    constexpr int NM = (P + 1) * (P + 2) * (P + 3) / 6;
    double C[NM], M[NM];
#pragma unroll
    for (int k = 0; k < NM; ++k) { C[k] = 0.0; M[k] = 0.0; }
    C[0] = m0;
    if (ORDER >= 2) {
        const CellM2 Q = cellM2[c];
        C[bidx(2, 0, 0)] = Q.xx; C[bidx(1, 1, 0)] = Q.xy; C[bidx(1, 0, 1)] = Q.xz; C[bidx(0, 2, 0)] = Q.yy; C[bidx(0, 1, 1)] = Q.yz; C[bidx(0, 0, 2)] = Q.zz;
    }
    if (ORDER >= 4) {
        const CellM34& R = cellM34[c];
#pragma unroll
        for (int k = 0; k < 25; ++k) C[10 + k] = R.v[k];
    }
    // M_abc = sum_{i<=a, j<=b, k<=c} C(a,i) C(b,j) C(c,k) C_ijk d^(a-i, b-j, c-k)  -  rhobar x (cube moment)
    double px[P + 1], py[P + 1], pz[P + 1];
    px[0] = py[0] = pz[0] = 1.0;
#pragma unroll
    for (int k = 1; k <= P; ++k) { px[k] = px[k - 1] * dx; py[k] = py[k - 1] * dy; pz[k] = pz[k - 1] * dz; }
#pragma unroll
    for (int d = 0; d <= P; ++d)
#pragma unroll
        for (int a = d; a >= 0; --a)
#pragma unroll
            for (int b = d - a; b >= 0; --b) {
                const int cc = d - a - b;
                double s = 0;
#pragma unroll
                for (int i = 0; i <= a; ++i)
#pragma unroll
                    for (int j = 0; j <= b; ++j)
#pragma unroll
                        for (int k = 0; k <= cc; ++k) {
                            double w = 1.0;
                            for (int t = 0; t < i; ++t) w = w * (a - t) / (t + 1);
                            for (int t = 0; t < j; ++t) w = w * (b - t) / (t + 1);
                            for (int t = 0; t < k; ++t) w = w * (cc - t) / (t + 1);
                            s += w * C[bidx(i, j, k)] * px[a - i] * py[b - j] * pz[cc - k];
                        }
                M[bidx(a, b, cc)] = s - rhobar * cube1d(a, side) * cube1d(b, side) * cube1d(cc, side);
            }
    bgA[c] = make_float4((float)M[0], (float)M[1], (float)M[2], (float)M[3]);
    if (ORDER >= 2) {
        CellM2 E;
        const float xx = (float)M[bidx(2, 0, 0)], xy = (float)M[bidx(1, 1, 0)], xz = (float)M[bidx(1, 0, 1)], yy = (float)M[bidx(0, 2, 0)],
                    yz = (float)M[bidx(0, 1, 1)], zz = (float)M[bidx(0, 0, 2)], t2 = xx + yy + zz;
        E.xx = 3.f * xx; E.xy = 3.f * xy; E.xz = 3.f * xz; E.yy = 3.f * yy; E.yz = 3.f * yz; E.zz = 3.f * zz; E.t2 = 1.5f * t2; E.pad1 = 0.5f * t2;
        bgE2[c] = E;
    }
    if (ORDER >= 4) {
        CellM34 R;
        float* v = R.v;
#pragma unroll
        for (int k = 0; k < 25; ++k) v[k] = (float)M[10 + k];
        const float* m3 = v; const float* m4 = v + 10;
        v[25] = m3[0] + m3[3] + m3[5]; v[26] = m3[1] + m3[6] + m3[8]; v[27] = m3[2] + m3[7] + m3[9];
        v[28] = m4[0] + m4[3] + m4[5]; v[29] = m4[1] + m4[6] + m4[8]; v[30] = m4[2] + m4[7] + m4[9];
        v[31] = m4[3] + m4[10] + m4[12]; v[32] = m4[4] + m4[11] + m4[13]; v[33] = m4[5] + m4[12] + m4[14];
        v[34] = v[28] + v[31] + v[33]; v[35] = 0.f;
        bgM34[c] = R;
    }
}

// potential (-int dy/|x-y|) and acceleration at the origin-shifted point of the homogeneous unit-density cube whose corners
// are (X0 or X0+side, ...) relative to the point; closed form, fp64 (the oracle's orc_cube_field restated)
__device__ __forceinline__ double cube_l(double a, double b, double c, double r) { return a * b == 0.0 ? 0.0 : a * b * log(c + r); }
__device__ __forceinline__ double cube_t(double a, double b, double c, double r) { return a == 0.0 ? 0.0 : 0.5 * a * a * atan(b * c / (a * r)); }
__device__ __forceinline__ double cube_d(double X, double Y, double Z, double r) {
    return (Y == 0.0 ? 0.0 : Y * log(Z + r)) + (Z == 0.0 ? 0.0 : Z * log(Y + r)) - (X == 0.0 ? 0.0 : X * atan(Y * Z / (X * r)));
}
__device__ void cube_field(double X0, double Y0, double Z0, double side, double w, double (&acc)[4]) { // acc += w x (ax, ay, az, phi)
    double f = 0, gx = 0, gy = 0, gz = 0;
    for (int i = 0; i < 2; ++i) for (int j = 0; j < 2; ++j) for (int k = 0; k < 2; ++k) {
        const double X = X0 + i * side, Y = Y0 + j * side, Z = Z0 + k * side, r = sqrt(X * X + Y * Y + Z * Z), sg = ((i + j + k) & 1) ? -1.0 : 1.0;
        f += sg * (cube_l(X, Y, Z, r) + cube_l(Y, Z, X, r) + cube_l(Z, X, Y, r) - cube_t(X, Y, Z, r) - cube_t(Y, Z, X, r) - cube_t(Z, X, Y, r));
        gx += sg * cube_d(X, Y, Z, r); gy += sg * cube_d(Y, Z, X, r); gz += sg * cube_d(Z, X, Y, r);
    }
    acc[0] += w * gx; acc[1] += w * gy; acc[2] += w * gz; acc[3] += w * f;
}

#define BG_WARPS 4
template <int ORDER>
__global__ void __launch_bounds__(BG_WARPS * 32) forces_bg_kernel(const __grid_constant__ ForceArgs A, const double* __restrict__ far, double* __restrict__ farc,
                                                                  const float4* __restrict__ bgA, const CellM2* __restrict__ bgE2, const CellM34* __restrict__ bgM34,
                                                                  const uint4* __restrict__ pvlist, const uint32_t* __restrict__ lpv, const unsigned long long* __restrict__ pvoff,
                                                                  double rhobar, int with_cells) {
    __shared__ __align__(16) float s_rec[BG_WARPS][4 + 4 + 8 + 36];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    float* const rec = s_rec[w];
    const double h = A.size * (1.0 / 2097152.0);
    for (int64_t gi = A.g0 + (int64_t)blockIdx.x * BG_WARPS + w; gi < A.g1; gi += (int64_t)gridDim.x * BG_WARPS) {
        const GroupRec g = A.group[gi];
        const WalkCell gw = A.wcell[g.cell];
        const int gs = 1 << (HOT_MAXLEVEL - (int)(gw.w >> 27));
        const int gox = (int)(gw.x & 0x1fffffu), goy = (int)((gw.x >> 21) | ((gw.y & 0x3ffu) << 11)), goz = (int)((gw.y >> 10) & 0x1fffffu);
        const double ox = A.lo[0] + ((double)gox + 0.5 * gs) * h, oy = A.lo[1] + ((double)goy + 0.5 * gs) * h, oz = A.lo[2] + ((double)goz + 0.5 * gs) * h;
        const unsigned long long o0 = A.pcoff[gi] + A.lpc0[gi]; // the flagged cells follow the plain ones
        const int n = with_cells ? (int)A.lpc2[gi] : 0, nv = (int)lpv[gi]; // with_cells = 0: the flagged cells go through hot_forces.cu's kernel
        const unsigned long long v0 = pvoff[gi];
        for (uint32_t s0 = 0; s0 < g.count; s0 += 32) {
            const uint32_t loc = s0 + lane;
            const bool on = loc < g.count;
            const float4 b = A.body[g.first + (on ? loc : 0u)];
            const float x[3] = {(float)((double)b.x - ox), (float)((double)b.y - oy), (float)((double)b.z - oz)};
            double S[4] = {0.0, 0.0, 0.0, 0.0};
            float a[4] = {0.f, 0.f, 0.f, 0.f};
            int nacc = 0;
            for (int j = 0; j < n + nv; ++j) {
                __syncwarp();
                if (j < n) { // a background-subtracted cell: its record, its centre shifted to its image
                    const uint32_t c = A.pclist[o0 + j] & 0x0fffffffu;
                    const int im = A.pcimg[o0 + j];
                    if (lane == 0) {
                        const WalkCell wc = A.wcell[c];
                        const double side = ldexp(A.size, -(int)(wc.w >> 27));
                        const double cx = A.lo[0] + (double)(wc.x & 0x1fffffu) * h + 0.5 * side + (double)(im / 25 - 2) * A.size;
                        const double cy = A.lo[1] + (double)((wc.x >> 21) | ((wc.y & 0x3ffu) << 11)) * h + 0.5 * side + (double)((im / 5) % 5 - 2) * A.size;
                        const double cz = A.lo[2] + (double)((wc.y >> 10) & 0x1fffffu) * h + 0.5 * side + (double)(im % 5 - 2) * A.size;
                        const float4 m = bgA[c];
                        rec[0] = (float)(ox - cx); rec[1] = (float)(oy - cy); rec[2] = (float)(oz - cz); rec[3] = -m.x;
                        rec[4] = m.y; rec[5] = m.z; rec[6] = m.w; rec[7] = 0.f;
                    }
                    if (ORDER >= 2 && lane < 8) rec[8 + lane] = reinterpret_cast<const float*>(bgE2 + c)[lane];
                    if (ORDER >= 4) { rec[16 + lane] = bgM34[c].v[lane]; if (lane < 4) rec[48 + lane] = bgM34[c].v[32 + lane]; }
                } else { // a virtual cube: minus the uniform cube's moments about its centre
                    const uint4 e = pvlist[v0 + (j - n)];
                    if (lane == 0) {
                        const int lev = (int)e.z, im = (int)e.w;
                        const double side = ldexp(A.size, -lev);
                        const double cx = A.lo[0] + (double)(e.x & 0x1fffffu) * h + 0.5 * side + (double)(im / 25 - 2) * A.size;
                        const double cy = A.lo[1] + (double)((e.x >> 21) | ((e.y & 0x3ffu) << 11)) * h + 0.5 * side + (double)((im / 5) % 5 - 2) * A.size;
                        const double cz = A.lo[2] + (double)((e.y >> 10) & 0x1fffffu) * h + 0.5 * side + (double)(im % 5 - 2) * A.size;
                        const double s2 = side * side, m0 = -rhobar * side * s2, m2 = m0 * s2 / 12.0, m4a = m0 * s2 * s2 / 80.0, m4b = m0 * s2 * s2 / 144.0;
                        rec[0] = (float)(ox - cx); rec[1] = (float)(oy - cy); rec[2] = (float)(oz - cz); rec[3] = (float)(-m0);
                        rec[4] = rec[5] = rec[6] = rec[7] = 0.f;
                        const float t2 = (float)(3.0 * m2);
                        rec[8] = (float)(3.0 * m2); rec[9] = 0.f; rec[10] = 0.f; rec[11] = (float)(3.0 * m2); rec[12] = 0.f; rec[13] = (float)(3.0 * m2); rec[14] = 1.5f * t2; rec[15] = 0.5f * t2;
                        for (int k = 0; k < 36; ++k) rec[16 + k] = 0.f;
                        // M4 (degree-major: xxxx xxxy xxxz xxyy xxyz xxzz xyyy xyyz xyzz xzzz yyyy yyyz yyzz yzzz zzzz)
                        float* m4 = rec + 16 + 10;
                        m4[0] = m4[10] = m4[14] = (float)m4a; m4[3] = m4[5] = m4[12] = (float)m4b;
                        float* v = rec + 16;
                        v[28] = m4[0] + m4[3] + m4[5]; v[31] = m4[3] + m4[10] + m4[12]; v[33] = m4[5] + m4[12] + m4[14]; v[34] = v[28] + v[31] + v[33];
                    }
                }
                __syncwarp();
                const float4 q0 = make_float4(rec[0], rec[1], rec[2], rec[3]);
                const float4 q1 = make_float4(rec[8], rec[9], rec[10], rec[11]), q2 = make_float4(rec[12], rec[13], rec[14], rec[15]);
                pc_one<ORDER, float>(q0, q1, q2, rec + 16, x, A.spline ? 0.f : A.eps2, a);
                { // the dipole term: phi_1 = D1 (M1 . R), a_1 = -[D2 (M1 . R) R + D1 M1], D1 = -u^-3/2, D2 = 3 u^-5/2
                    const float Rx = x[0] + q0.x, Ry = x[1] + q0.y, Rz = x[2] + q0.z;
                    const float ri = rsqrt_approx(fmaf(Rx, Rx, fmaf(Ry, Ry, fmaf(Rz, Rz, A.spline ? 0.f : A.eps2)))), ri3 = ri * ri * ri;
                    const float dR = fmaf(rec[4], Rx, fmaf(rec[5], Ry, rec[6] * Rz)), c5 = -3.0f * ri3 * ri * ri * dR;
                    a[0] += fmaf(c5, Rx, ri3 * rec[4]); a[1] += fmaf(c5, Ry, ri3 * rec[5]); a[2] += fmaf(c5, Rz, ri3 * rec[6]);
                    a[3] -= ri3 * dR;
                }
                if (++nacc == 64) { S[0] += (double)a[0]; S[1] += (double)a[1]; S[2] += (double)a[2]; S[3] += (double)a[3]; a[0] = a[1] = a[2] = a[3] = 0.f; nacc = 0; }
            }
            S[0] += (double)a[0]; S[1] += (double)a[1]; S[2] += (double)a[2]; S[3] += (double)a[3];
            if (on) {
                // what was subtracted, added back in closed form (fp64): rhobar x [homogeneous (5 L)^3 cube - homogeneous K_G]
                cube_field(A.lo[0] - 2.0 * A.size - (double)b.x, A.lo[1] - 2.0 * A.size - (double)b.y, A.lo[2] - 2.0 * A.size - (double)b.z, 5.0 * A.size, rhobar, S);
                cube_field(A.lo[0] + (double)(gox - 2 * gs) * h - (double)b.x, A.lo[1] + (double)(goy - 2 * gs) * h - (double)b.y,
                           A.lo[2] + (double)(goz - 2 * gs) * h - (double)b.z, 5.0 * (double)gs * h, -rhobar, S);
                const double4 f = reinterpret_cast<const double4*>(far)[g.first + loc];
                double4 r; r.x = f.x + S[0]; r.y = f.y + S[1]; r.z = f.z + S[2]; r.w = f.w + S[3];
                reinterpret_cast<double4*>(farc)[g.first + loc] = r;
            }
        }
    }
}

cudaError_t launch_bg_moments(const Tree& t, int order, double rhobar, cudaStream_t st) {
    const unsigned nb = (unsigned)((t.ncells + 127) / 128);
    HOT_LAUNCHED(1);
    if (order >= 4) bg_moments_kernel<4><<<nb, 128, 0, st>>>(t.wcell, t.cellA, t.cellM0d, t.cellM2, t.cellM34, t.ncells, t.lo[0], t.lo[1], t.lo[2], t.size, rhobar, t.bgA, t.bgE2, t.bgM34);
    else if (order >= 2) bg_moments_kernel<2><<<nb, 128, 0, st>>>(t.wcell, t.cellA, t.cellM0d, t.cellM2, t.cellM34, t.ncells, t.lo[0], t.lo[1], t.lo[2], t.size, rhobar, t.bgA, t.bgE2, t.bgM34);
    else bg_moments_kernel<0><<<nb, 128, 0, st>>>(t.wcell, t.cellA, t.cellM0d, t.cellM2, t.cellM34, t.ncells, t.lo[0], t.lo[1], t.lo[2], t.size, rhobar, t.bgA, t.bgE2, t.bgM34);
    return cudaGetLastError();
}
cudaError_t launch_forces_bg(const ForceArgs& a, const Tree& t, const double* far, double* farc, const uint4* pvlist, const uint32_t* lpv,
                             const unsigned long long* pvoff, double rhobar, int with_cells, cudaStream_t st) {
    const int64_t ng = a.g1 - a.g0;
    if (ng <= 0) return cudaSuccess;
    int64_t nb = (ng + BG_WARPS - 1) / BG_WARPS;
    if (nb > 148 * 32) nb = 148 * 32;
    HOT_LAUNCHED(1);
    if (a.order >= 4) forces_bg_kernel<4><<<(unsigned)nb, BG_WARPS * 32, 0, st>>>(a, far, farc, t.bgA, t.bgE2, t.bgM34, pvlist, lpv, pvoff, rhobar, with_cells);
    else if (a.order >= 2) forces_bg_kernel<2><<<(unsigned)nb, BG_WARPS * 32, 0, st>>>(a, far, farc, t.bgA, t.bgE2, t.bgM34, pvlist, lpv, pvoff, rhobar, with_cells);
    else forces_bg_kernel<0><<<(unsigned)nb, BG_WARPS * 32, 0, st>>>(a, far, farc, t.bgA, t.bgE2, t.bgM34, pvlist, lpv, pvoff, rhobar, with_cells);
    return cudaGetLastError();
}

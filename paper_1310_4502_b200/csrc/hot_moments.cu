// hot_moments.cu -- S6 upward pass: mass, centre of mass and raw Cartesian moments of eq (6)
// about the centre of mass, per cell, level by level from the leaves up.
// Leaves sum their bodies; internal cells combine their children with the parallel-axis shift
//   M'_alpha = sum_{beta<=alpha} C(alpha,beta) M_beta d^(alpha-beta),  d = z_child - z_parent.
// Arithmetic is fp64 (the stage is HBM/latency bound); results are stored as the fp32 records the
// interaction kernels stage, except the centre of mass which stays fp64.
#include "hot_internal.h"

// multi-index (a,b,c) -> position, degree-major, x>y>z (same enumeration the moments are exported in)
__host__ __device__ constexpr int midx(int a, int b, int c) {
    int d = a + b + c;
    return d * (d + 1) * (d + 2) / 6 + (d - a) * (d - a + 1) / 2 + (d - a - b);
}
template <int ORDER> struct NMom { static constexpr int v = (ORDER >= 4) ? 35 : (ORDER >= 2 ? 10 : 4); };

template <int ORDER>
__device__ __forceinline__ void add_point(double* M, double m, double dx, double dy, double dz) {
    // M[midx(a,b,c)] += m dx^a dy^b dz^c for 2 <= a+b+c <= ORDER
    constexpr int P = ORDER >= 4 ? 4 : 2;
    double px[P + 1], py[P + 1], pz[P + 1];
    px[0] = py[0] = pz[0] = 1.0;
#pragma unroll
    for (int k = 1; k <= P; ++k) { px[k] = px[k - 1] * dx; py[k] = py[k - 1] * dy; pz[k] = pz[k - 1] * dz; }
#pragma unroll
    for (int d = 2; d <= P; ++d)
#pragma unroll
        for (int a = d; a >= 0; --a)
#pragma unroll
            for (int b = d - a; b >= 0; --b) M[midx(a, b, d - a - b)] += m * px[a] * py[b] * pz[d - a - b];
}
__host__ __device__ constexpr double binom_c(int n, int k) {
    double r = 1;
    for (int i = 0; i < k; ++i) r = r * (n - i) / (i + 1);
    return r;
}
// out += shift of child moments C (about its own centre, dipole = 0) by d
template <int ORDER>
__device__ __forceinline__ void add_shifted(double* M, const double* C, double m0, double dx, double dy, double dz) {
    constexpr int P = ORDER >= 4 ? 4 : 2;
    double px[P + 1], py[P + 1], pz[P + 1];
    px[0] = py[0] = pz[0] = 1.0;
#pragma unroll
    for (int k = 1; k <= P; ++k) { px[k] = px[k - 1] * dx; py[k] = py[k - 1] * dy; pz[k] = pz[k - 1] * dz; }
#pragma unroll
    for (int d = 2; d <= P; ++d)
#pragma unroll
        for (int a = d; a >= 0; --a)
#pragma unroll
            for (int b = d - a; b >= 0; --b) {
                const int c = d - a - b;
                double s = 0;
#pragma unroll
                for (int i = 0; i <= a; ++i)
#pragma unroll
                    for (int j = 0; j <= b; ++j)
#pragma unroll
                        for (int k = 0; k <= c; ++k) {
                            const int e = i + j + k;
                            if (e == 1) continue; // dipole about the child's centre of mass
                            const double w = binom_c(a, i) * binom_c(b, j) * binom_c(c, k);
                            const double mb = e == 0 ? m0 : C[midx(i, j, k)];
                            s += w * mb * px[a - i] * py[b - j] * pz[c - k];
                        }
                M[midx(a, b, c)] += s;
            }
}

template <int ORDER>
__device__ __forceinline__ void store_cell(int64_t c, double m0, double zx, double zy, double zz, double bmax, const double* M,
                                           CellA* cellA, CellM2* cellM2, CellM2* cellE2, CellM34* cellM34) {
    CellA A; A.zx = zx; A.zy = zy; A.zz = zz; A.m0 = (float)m0; A.bmax = __double2float_ru(bmax); // rounded up: stays a bound
    if (ORDER >= 2) {
        CellM2 Q;
        Q.xx = (float)M[midx(2, 0, 0)]; Q.xy = (float)M[midx(1, 1, 0)]; Q.xz = (float)M[midx(1, 0, 1)];
        Q.yy = (float)M[midx(0, 2, 0)]; Q.yz = (float)M[midx(0, 1, 1)]; Q.zz = (float)M[midx(0, 0, 2)];
        const float t2 = Q.xx + Q.yy + Q.zz;
        Q.t2 = t2; Q.pad1 = 0.f;
        cellM2[c] = Q;
        CellM2 E; // what the P-C kernel stages: phi2 = 0.5 t2 ri^3 - 0.5 ri^5 R.(3 M2).R, a2 = R (1.5 t2 ri^5 - 2.5 ri^7 R.(3 M2).R) + ri^5 (3 M2) R
        E.xx = 3.f * Q.xx; E.xy = 3.f * Q.xy; E.xz = 3.f * Q.xz; E.yy = 3.f * Q.yy; E.yz = 3.f * Q.yz; E.zz = 3.f * Q.zz;
        E.t2 = 1.5f * t2; E.pad1 = 0.5f * t2;
        cellE2[c] = E;
    }
    cellA[c] = A;
    if (ORDER >= 4) {
        CellM34 R;
        float* v = R.v;
#pragma unroll
        for (int k = 0; k < 25; ++k) v[k] = (float)M[10 + k]; // M3 (10) then M4 (15), degree-major
        const float* m3 = v; const float* m4 = v + 10;
        // traces: t3_k = M3_iik, T4_kl = M4_iikl, t4 = M4_iijj
        v[25] = m3[0] + m3[3] + m3[5];                 // xxx + xyy + xzz
        v[26] = m3[1] + m3[6] + m3[8];                 // xxy + yyy + yzz
        v[27] = m3[2] + m3[7] + m3[9];                 // xxz + yyz + zzz
        v[28] = m4[0] + m4[3] + m4[5];                 // T4xx = xxxx + xxyy + xxzz
        v[29] = m4[1] + m4[6] + m4[8];                 // T4xy = xxxy + xyyy + xyzz
        v[30] = m4[2] + m4[7] + m4[9];                 // T4xz = xxxz + xyyz + xzzz
        v[31] = m4[3] + m4[10] + m4[12];               // T4yy = xxyy + yyyy + yyzz
        v[32] = m4[4] + m4[11] + m4[13];               // T4yz = xxyz + yyyz + yzzz
        v[33] = m4[5] + m4[12] + m4[14];               // T4zz = xxzz + yyzz + zzzz
        v[34] = v[28] + v[31] + v[33];                 // t4
        v[35] = 0.f;
        cellM34[c] = R;
    }
}
template <int ORDER>
__device__ __forceinline__ void load_child(int64_t c, const CellA* cellA, const CellM2* cellM2, const CellM34* cellM34, double* C) {
    if (ORDER >= 2) {
        CellM2 Q = cellM2[c];
        C[midx(2, 0, 0)] = Q.xx; C[midx(1, 1, 0)] = Q.xy; C[midx(1, 0, 1)] = Q.xz;
        C[midx(0, 2, 0)] = Q.yy; C[midx(0, 1, 1)] = Q.yz; C[midx(0, 0, 2)] = Q.zz;
    }
    if (ORDER >= 4) {
        const CellM34& R = cellM34[c];
#pragma unroll
        for (int k = 0; k < 25; ++k) C[10 + k] = R.v[k];
    }
}

template <int ORDER>
__global__ void __launch_bounds__(128) moments_level_kernel(int64_t cbeg, int64_t cend, const uint32_t* __restrict__ cfirst,
                                                            const uint32_t* __restrict__ ccount, const uint32_t* __restrict__ cmask,
                                                            const int32_t* __restrict__ cchild, const float4* __restrict__ body,
                                                            CellA* __restrict__ cellA, CellM2* __restrict__ cellM2, CellM2* __restrict__ cellE2,
                                                            CellM34* __restrict__ cellM34) {
    int64_t c = cbeg + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= cend) return;
    constexpr int NM = NMom<ORDER>::v;
    double M[NM];
#pragma unroll
    for (int k = 0; k < NM; ++k) M[k] = 0;
    double m0 = 0, zx = 0, zy = 0, zz = 0, bmax = 0; // bmax: DESIGN.md R-15 (leaf: farthest body; else children's radii + offsets)
    int32_t ch = cchild[c];
    if (ch < 0) { // leaf: from its bodies
        uint32_t f = cfirst[c], n = ccount[c];
        for (uint32_t j = 0; j < n; ++j) {
            float4 b = body[f + j];
            m0 += (double)b.w; zx += (double)b.w * b.x; zy += (double)b.w * b.y; zz += (double)b.w * b.z;
        }
        zx /= m0; zy /= m0; zz /= m0;
        for (uint32_t j = 0; j < n; ++j) {
            float4 b = body[f + j];
            const double dx = (double)b.x - zx, dy = (double)b.y - zy, dz = (double)b.z - zz;
            bmax = fmax(bmax, dx * dx + dy * dy + dz * dz);
            if (ORDER >= 2) add_point<ORDER>(M, (double)b.w, dx, dy, dz);
        }
        bmax = sqrt(bmax);
    } else { // internal: from its children (one level down, already done)
        int nch = __popc(cmask[c]);
        for (int k = 0; k < nch; ++k) {
            CellA A = cellA[ch + k];
            m0 += (double)A.m0; zx += (double)A.m0 * A.zx; zy += (double)A.m0 * A.zy; zz += (double)A.m0 * A.zz;
        }
        zx /= m0; zy /= m0; zz /= m0;
        for (int k = 0; k < nch; ++k) {
            CellA A = cellA[ch + k];
            const double dx = A.zx - zx, dy = A.zy - zy, dz = A.zz - zz;
            bmax = fmax(bmax, sqrt(dx * dx + dy * dy + dz * dz) + (double)A.bmax);
            if (ORDER >= 2) {
                double C[NM];
                load_child<ORDER>(ch + k, cellA, cellM2, cellM34, C);
                add_shifted<ORDER>(M, C, (double)A.m0, dx, dy, dz);
            }
        }
    }
    store_cell<ORDER>(c, m0, zx, zy, zz, bmax, M, cellA, cellM2, cellE2, cellM34);
}

cudaError_t launch_moments(const Tree& t, int order, cudaStream_t st) {
    for (int l = t.max_level; l >= 0; --l) {
        int64_t cb = t.level_base[l], ce = t.level_base[l + 1];
        if (ce <= cb) continue;
        unsigned nb = (unsigned)((ce - cb + 127) / 128);
        HOT_LAUNCHED(1);
        if (order >= 4)
            moments_level_kernel<4><<<nb, 128, 0, st>>>(cb, ce, t.cfirst, t.ccount, t.cmask, t.cchild, t.body, t.cellA, t.cellM2, t.cellE2, t.cellM34);
        else if (order >= 2)
            moments_level_kernel<2><<<nb, 128, 0, st>>>(cb, ce, t.cfirst, t.ccount, t.cmask, t.cchild, t.body, t.cellA, t.cellM2, t.cellE2, t.cellM34);
        else
            moments_level_kernel<0><<<nb, 128, 0, st>>>(cb, ce, t.cfirst, t.ccount, t.cmask, t.cchild, t.body, t.cellA, t.cellM2, t.cellE2, t.cellM34);
    }
    return cudaGetLastError();
}

// hot_moments.cu -- S6 upward pass: mass, centre of mass, raw Cartesian moments of eq (6)
// about the centre of mass and b_max, per cell, from the leaves up.
// Leaves sum their bodies; internal cells combine their children with the parallel-axis shift
//   M'_alpha = sum_{beta<=alpha} C(alpha,beta) M_beta d^(alpha-beta),  d = z_child - z_parent.
// Arithmetic is fp64 (the stage is HBM/latency bound); results are stored as the fp32 records the
// interaction kernels stage, except the centre of mass which stays fp64.
#include "hot_internal.h"
#include "hot_hi_generated.inc" // f-3: record layouts and builders of the orders 6 and 8 (gen_hi_orders.py)

// multi-index (a,b,c) -> position, degree-major, x>y>z (same enumeration the moments are exported in)
__host__ __device__ constexpr int midx(int a, int b, int c) {
    int d = a + b + c;
    return d * (d + 1) * (d + 2) / 6 + (d - a) * (d - a + 1) / 2 + (d - a - b);
}
template <int ORDER> struct NMom { static constexpr int v = ORDER >= 2 ? (ORDER + 1) * (ORDER + 2) * (ORDER + 3) / 6 : 4; }; // 10, 35, 84, 165

template <int ORDER>
__device__ __forceinline__ void add_point(double* M, double m, double dx, double dy, double dz) {
    // M[midx(a,b,c)] += m dx^a dy^b dz^c for 2 <= a+b+c <= ORDER
    constexpr int P = ORDER >= 4 ? ORDER : 2;
    if constexpr (ORDER > 4) { // orders 6, 8 (f-3): plain loops -- 165 moments unrolled would take ptxas many minutes
        double px[P + 1], py[P + 1], pz[P + 1];
        px[0] = py[0] = pz[0] = 1.0;
        for (int k = 1; k <= P; ++k) { px[k] = px[k - 1] * dx; py[k] = py[k - 1] * dy; pz[k] = pz[k - 1] * dz; }
#pragma unroll 1
        for (int d = 2; d <= P; ++d)
#pragma unroll 1
            for (int a = d; a >= 0; --a)
#pragma unroll 1
                for (int b = d - a; b >= 0; --b) M[midx(a, b, d - a - b)] += m * px[a] * py[b] * pz[d - a - b];
        return;
    }
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
    constexpr int P = ORDER >= 4 ? ORDER : 2;
    if constexpr (ORDER > 4) { // plain loops, as in add_point
        double px[P + 1], py[P + 1], pz[P + 1], bin[P + 1][P + 1];
        px[0] = py[0] = pz[0] = 1.0;
        for (int k = 1; k <= P; ++k) { px[k] = px[k - 1] * dx; py[k] = py[k - 1] * dy; pz[k] = pz[k - 1] * dz; }
        for (int n = 0; n <= P; ++n) { bin[n][0] = 1.0; for (int k = 1; k <= n; ++k) bin[n][k] = bin[n][k - 1] * (double)(n - k + 1) / (double)k; }
#pragma unroll 1
        for (int d = 2; d <= P; ++d)
#pragma unroll 1
            for (int a = d; a >= 0; --a)
#pragma unroll 1
                for (int b = d - a; b >= 0; --b) {
                    const int c = d - a - b;
                    double s = 0;
#pragma unroll 1
                    for (int i = 0; i <= a; ++i)
#pragma unroll 1
                        for (int j = 0; j <= b; ++j)
#pragma unroll 1
                            for (int k = 0; k <= c; ++k) {
                                const int e = i + j + k;
                                if (e == 1) continue; // dipole about the child's centre of mass
                                const double mb = e == 0 ? m0 : C[midx(i, j, k)];
                                s += bin[a][i] * bin[b][j] * bin[c][k] * mb * px[a - i] * py[b - j] * pz[c - k];
                            }
                    M[midx(a, b, c)] += s;
                }
        return;
    }
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
                                           CellA* cellA, CellM2* cellM2, CellM2* cellE2, CellM34* cellM34, float4* cellMac = nullptr,
                                           float* hiRaw = nullptr, float* hiT = nullptr, double side = 1.0) {
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
        if constexpr (ORDER > 4) { // f-3: degrees 5 .. ORDER, in units of the cell's side (fp32 range), raw and as the trace record
            constexpr int NRAW = HiOrder<ORDER>::NRAW, NT = HiOrder<ORDER>::NT;
            const double inv = 1.0 / side;
            double sc = inv * inv * inv * inv;
            int k = 35;
#pragma unroll 1
            for (int d = 5; d <= ORDER; ++d) {
                sc *= inv;
#pragma unroll 1
                for (int q = 0; q < (d + 1) * (d + 2) / 2; ++q, ++k) hiRaw[(size_t)c * NRAW + (k - 35)] = (float)(M[k] * sc);
            }
            hi_record<ORDER>(M, inv, hiT + (size_t)c * NT);
        }
        if (cellMac) { // numerators of the error bounds of DESIGN.md R-16, rounded up: b, 3 B2, 4 sqrt(B2 B4), 6 b B4
            const double B2 = M[midx(2, 0, 0)] + M[midx(0, 2, 0)] + M[midx(0, 0, 2)];
            const double B4 = M[midx(4, 0, 0)] + M[midx(0, 4, 0)] + M[midx(0, 0, 4)] + 2.0 * (M[midx(2, 2, 0)] + M[midx(2, 0, 2)] + M[midx(0, 2, 2)]);
            cellMac[c] = make_float4(A.bmax, __double2float_ru(3.0 * B2), __double2float_ru(4.0 * sqrt(B2 * B4)), __double2float_ru(6.0 * (double)A.bmax * B4));
        }
    }
}
template <int ORDER>
__device__ __forceinline__ void load_child(int64_t c, const CellM2* cellM2, const CellM34* cellM34, double* C, const float* hiRaw = nullptr, double side = 1.0) {
    if (ORDER >= 2) {
        const float4 q0 = reinterpret_cast<const float4*>(cellM2 + c)[0], q1 = reinterpret_cast<const float4*>(cellM2 + c)[1];
        C[midx(2, 0, 0)] = q0.x; C[midx(1, 1, 0)] = q0.y; C[midx(1, 0, 1)] = q0.z;
        C[midx(0, 2, 0)] = q0.w; C[midx(0, 1, 1)] = q1.x; C[midx(0, 0, 2)] = q1.y;
    }
    if (ORDER >= 4) {
        const float4* r = reinterpret_cast<const float4*>(cellM34 + c);
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const float4 v = r[k];
            C[10 + 4 * k] = v.x; C[11 + 4 * k] = v.y; C[12 + 4 * k] = v.z; C[13 + 4 * k] = v.w;
        }
        C[34] = reinterpret_cast<const float*>(cellM34 + c)[24];
    }
    if constexpr (ORDER > 4) {
        constexpr int NRAW = HiOrder<ORDER>::NRAW;
        double sc = side * side * side * side;
        int k = 35;
#pragma unroll 1
        for (int d = 5; d <= ORDER; ++d) {
            sc *= side;
#pragma unroll 1
            for (int q = 0; q < (d + 1) * (d + 2) / 2; ++q, ++k) C[k] = (double)hiRaw[(size_t)c * NRAW + (k - 35)] * sc;
        }
    }
}

// Leaves, one thread each, in BODY order (leafcell, written by tree_emit): neighbouring threads read neighbouring
// bodies (a leaf holds 4 bodies on average at NLEAF = 16, so the lines a warp touches are shared through L1).
struct MomArgs {
    const int32_t* leafcell; int64_t nleaves;
    const uint32_t *cfirst, *ccount, *cmask; const int32_t* cchild; const float4* body;
    CellA* cellA; CellM2* cellM2; CellM2* cellE2; CellM34* cellM34; float4* cellMac;
    double* m0d; // periodic boxes: the cell mass in fp64 (the background-subtracted mass of hot_bg.cu is a small difference), else NULL
    float *hiRaw, *hiT; const WalkCell* wcell; double size; // orders 6, 8: raw and trace records in units of the cell side (side = size / 2^level)
};
__device__ __forceinline__ double cell_side(const MomArgs& P, int64_t c) { return ldexp(P.size, -(int)(P.wcell[c].w >> 27)); }
template <int ORDER>
__global__ void __launch_bounds__(128) moments_leaves_kernel(const __grid_constant__ MomArgs P) {
    constexpr int NM = NMom<ORDER>::v;
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= P.nleaves) return;
    const int32_t c0 = P.leafcell[k];
    const uint32_t f = P.cfirst[c0], n = P.ccount[c0];
    double M[NM];
#pragma unroll
    for (int q = 0; q < NM; ++q) M[q] = 0;
    double m0 = 0, zx = 0, zy = 0, zz = 0, bmax = 0; // bmax: DESIGN.md R-15 (leaf: its farthest body)
    const float4* const src = P.body + f;
    for (uint32_t j = 0; j < n; ++j) {
        const float4 b = __ldg(src + j);
        m0 += (double)b.w; zx += (double)b.w * b.x; zy += (double)b.w * b.y; zz += (double)b.w * b.z;
    }
    zx /= m0; zy /= m0; zz /= m0;
    for (uint32_t j = 0; j < n; ++j) {
        const float4 b = __ldg(src + j);
        const double dx = (double)b.x - zx, dy = (double)b.y - zy, dz = (double)b.z - zz;
        bmax = fmax(bmax, dx * dx + dy * dy + dz * dz);
        if (ORDER >= 2) add_point<ORDER>(M, (double)b.w, dx, dy, dz);
    }
    if (P.m0d) P.m0d[c0] = m0;
    store_cell<ORDER>(c0, m0, zx, zy, zz, sqrt(bmax), M, P.cellA, P.cellM2, P.cellE2, P.cellM34, P.cellMac, P.hiRaw, P.hiT, ORDER > 4 ? cell_side(P, c0) : 1.0);
}
// an internal cell from its children (one level down, already done): parallel-axis shift, fixed child order
template <int ORDER>
__device__ __forceinline__ void combine_children(const MomArgs& P, int64_t c) {
    constexpr int NM = NMom<ORDER>::v;
    const int32_t ch = P.cchild[c];
    if (ch < 0) return; // a leaf: done by moments_leaves_kernel
    const int nch = __popc(P.cmask[c]);
    double M[NM];
#pragma unroll
    for (int q = 0; q < NM; ++q) M[q] = 0;
    double m0 = 0, zx = 0, zy = 0, zz = 0, bmax = 0; // bmax: DESIGN.md R-15 (children's radii + centre offsets)
    for (int q = 0; q < nch; ++q) {
        const CellA A = P.cellA[ch + q];
        const double cm = P.m0d ? P.m0d[ch + q] : (double)A.m0; // periodic boxes carry the masses in fp64 (a 2^24-body cell's mass does not fit fp32's 24 bits)
        m0 += cm; zx += cm * A.zx; zy += cm * A.zy; zz += cm * A.zz;
    }
    zx /= m0; zy /= m0; zz /= m0;
    for (int q = 0; q < nch; ++q) {
        const CellA A = P.cellA[ch + q];
        const double dx = A.zx - zx, dy = A.zy - zy, dz = A.zz - zz;
        bmax = fmax(bmax, sqrt(dx * dx + dy * dy + dz * dz) + (double)A.bmax);
        if (ORDER >= 2) {
            double C[NM];
            load_child<ORDER>(ch + q, P.cellM2, P.cellM34, C, P.hiRaw, ORDER > 4 ? cell_side(P, ch + q) : 1.0);
            add_shifted<ORDER>(M, C, P.m0d ? P.m0d[ch + q] : (double)A.m0, dx, dy, dz);
        }
    }
    if (P.m0d) P.m0d[c] = m0;
    store_cell<ORDER>(c, m0, zx, zy, zz, bmax, M, P.cellA, P.cellM2, P.cellE2, P.cellM34, P.cellMac, P.hiRaw, P.hiT, ORDER > 4 ? cell_side(P, c) : 1.0);
}
// One level of internal cells.  A warp looks at 32 consecutive cells of the level, keeps the internal ones (one in eight
// on average) and hands each to an OCTET of lanes: lane q of the octet loads child q (all children of the warp's cells in
// parallel instead of one dependent load chain per cell), the octet sums mass and centre of mass by shuffles, every lane
// shifts its child's moments to the parent's centre, and the octet sums them.  Four cells per trip.
template <int ORDER>
__global__ void __launch_bounds__(128) moments_level_kernel(const __grid_constant__ MomArgs P, int64_t cbeg, int64_t cend) {
    constexpr int NM = NMom<ORDER>::v;
    const int lane = threadIdx.x & 31, oct = lane >> 3, q = lane & 7;
    const int64_t c = cbeg + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int32_t ch0 = c < cend ? P.cchild[c] : -1;
    uint32_t todo = __ballot_sync(0xffffffffu, ch0 >= 0);
    const uint32_t mymask = ch0 >= 0 ? P.cmask[c] : 0u;
    while (todo) { // warp-uniform
        // the octet's cell: the oct-th set bit of todo
        uint32_t t = todo;
        for (int i = 0; i < oct; ++i) t &= t - 1;
        const int src = t ? __ffs((int)t) - 1 : 0;
        const bool have = t != 0;
        const int32_t ch = __shfl_sync(0xffffffffu, ch0, src);
        const int nch = __popc(__shfl_sync(0xffffffffu, mymask, src));
        const int64_t cell = (c - lane) + src;
        const bool mine = have && q < nch;
        CellA A; A.zx = A.zy = A.zz = 0.0; A.m0 = 0.f; A.bmax = 0.f;
        if (mine) A = P.cellA[ch + q];
        const double cm = mine ? (P.m0d ? P.m0d[ch + q] : (double)A.m0) : 0.0;
        double m0 = cm, zx = m0 * A.zx, zy = m0 * A.zy, zz = m0 * A.zz;
#pragma unroll
        for (int o = 1; o < 8; o <<= 1) {
            m0 += __shfl_xor_sync(0xffffffffu, m0, o); zx += __shfl_xor_sync(0xffffffffu, zx, o);
            zy += __shfl_xor_sync(0xffffffffu, zy, o); zz += __shfl_xor_sync(0xffffffffu, zz, o);
        }
        zx /= m0; zy /= m0; zz /= m0;
        double M[NM];
#pragma unroll
        for (int k = 0; k < NM; ++k) M[k] = 0;
        double bmax = 0; // DESIGN.md R-15: children's radii + centre offsets
        if (mine) {
            const double dx = A.zx - zx, dy = A.zy - zy, dz = A.zz - zz;
            bmax = sqrt(dx * dx + dy * dy + dz * dz) + (double)A.bmax;
            if (ORDER >= 2) {
                double C[NM];
                load_child<ORDER>(ch + q, P.cellM2, P.cellM34, C, P.hiRaw, ORDER > 4 ? cell_side(P, ch + q) : 1.0);
                add_shifted<ORDER>(M, C, cm, dx, dy, dz);
            }
        }
#pragma unroll
        for (int o = 1; o < 8; o <<= 1) {
            bmax = fmax(bmax, __shfl_xor_sync(0xffffffffu, bmax, o));
            if (ORDER >= 2) {
#pragma unroll
                for (int k = 4; k < NM; ++k) M[k] += __shfl_xor_sync(0xffffffffu, M[k], o);
            }
        }
        if (have && q == 0 && P.m0d) P.m0d[cell] = m0;
        if (have && q == 0) store_cell<ORDER>(cell, m0, zx, zy, zz, bmax, M, P.cellA, P.cellM2, P.cellE2, P.cellM34, P.cellMac, P.hiRaw, P.hiT, ORDER > 4 ? cell_side(P, cell) : 1.0);
        // drop the four cells just done
        for (int i = 0; i < 4 && todo; ++i) todo &= todo - 1;
    }
}
// the shallow levels ltop .. 0 (a few thousand cells in all) in one block: no launch per level
struct LevelBases { int64_t v[HOT_NLEVELS + 1]; };
template <int ORDER>
__global__ void __launch_bounds__(256) moments_top_kernel(const __grid_constant__ MomArgs P, const __grid_constant__ LevelBases LB, int ltop) {
    for (int l = ltop; l >= 0; --l) {
        for (int64_t c = LB.v[l] + threadIdx.x; c < LB.v[l + 1]; c += blockDim.x) combine_children<ORDER>(P, c);
        __syncthreads(); // this block wrote the level: visible to its own threads after the barrier
    }
}

template <int ORDER> static cudaError_t moments_run(const Tree& t, const MomArgs& a, cudaStream_t st) {
    HOT_LAUNCHED(1);
    moments_leaves_kernel<ORDER><<<(unsigned)((t.nleaves + 127) / 128), 128, 0, st>>>(a);
    // deepest level such that levels 0 .. ltop are cheap enough for ONE block (the order-4 shift is ~2000 fp64 operations per child)
    const int64_t top_cells = ORDER >= 6 ? 16 : ORDER >= 4 ? 128 : 640;
    int ltop = -1;
    while (ltop + 1 <= t.max_level && t.level_base[ltop + 2] <= top_cells) ++ltop;
    for (int l = t.max_level - 1; l > ltop; --l) { // the deepest level holds leaves only
        const int64_t cb = t.level_base[l], ce = t.level_base[l + 1];
        if (ce <= cb) continue;
        HOT_LAUNCHED(1);
        moments_level_kernel<ORDER><<<(unsigned)((ce - cb + 127) / 128), 128, 0, st>>>(a, cb, ce);
    }
    if (ltop >= 0) {
        LevelBases LB;
        for (int l = 0; l <= HOT_NLEVELS; ++l) LB.v[l] = t.level_base[l];
        HOT_LAUNCHED(1);
        moments_top_kernel<ORDER><<<1, 256, 0, st>>>(a, LB, ltop < t.max_level ? ltop : t.max_level);
    }
    return cudaGetLastError();
}
cudaError_t launch_moments(const Tree& t, int order, cudaStream_t st) {
    MomArgs a;
    a.leafcell = t.leafcell; a.nleaves = t.nleaves; a.cfirst = t.cfirst; a.ccount = t.ccount; a.cmask = t.cmask; a.cchild = t.cchild;
    a.body = t.body; a.cellA = t.cellA; a.cellM2 = t.cellM2; a.cellE2 = t.cellE2; a.cellM34 = t.cellM34; a.cellMac = order >= 4 ? t.cellMac : nullptr;
    a.hiRaw = t.cellHiRaw; a.hiT = t.cellHiT; a.wcell = t.wcell; a.size = t.size; a.m0d = t.cellM0d;
    if (order >= 8) return moments_run<8>(t, a, st);
    if (order >= 6) return moments_run<6>(t, a, st);
    if (order >= 4) return moments_run<4>(t, a, st);
    if (order >= 2) return moments_run<2>(t, a, st);
    return moments_run<0>(t, a, st);
}

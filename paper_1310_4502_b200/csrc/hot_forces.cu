// hot_forces.cu -- S8 particle-particle and S9 particle-cell interaction kernels, S10 scatter.
//
// Input: the interaction lists hot_walk.cu wrote for a range of sink groups (cell indices, body
// indices, image ids when periodic).  One warp owns one sink group at a time (persistent grid,
// dynamic group counter) and evaluates its lists in the m x n blocking of PAPER.md:162-164:
//
//   The 32 lanes are split into K = 32/L "source streams" of L lanes.  Every stream holds ALL sinks
//   of the group in registers (S = ceil(n/L) <= SMAX = 6 per lane) and takes every K-th source of a
//   32-source batch, read from shared memory as broadcast 128-bit loads.  L is the smallest power of
//   two with ceil(n/L) <= SMAX, so at most L-1 of the L*S sink slots idle whatever the group size;
//   the K partial sums are combined with shuffles once per group.
//
//   Batches are staged ahead of the arithmetic: list entries are read two batches ahead, cell
//   centres and bodies one batch ahead into registers (they need the fp64 shift to group-relative
//   coordinates), moments go global -> shared directly with cp.async (double-buffered).
//
// Arithmetic: interactions in fp32 (FFMA + MUFU.RSQ), coordinates relative to the group centre
// (formed in fp64 when a source is staged), per-lane partial sums of <= ~32 sources in fp32, running
// sums in fp64 (shared memory, lane-private).
#include "hot_internal.h"

#define FULL 0xffffffffu
#define BATCH 32               // sources per staged batch
#define WARPS_PER_BLOCK 4      // 3 blocks per SM at 166 registers (5 warps at 128 registers measured slower)
#define FLUSH_N 64             // sources a lane sums in fp32 before the partial sums go to the fp64 running sums
#define SMAX 6                 // sinks per lane (measured: 6 at 3 blocks/SM beats 4 at 4 and 8 at 2, NCRIT >= 128)
#define UNROLL2_S 6            // two sources per loop trip for this many sinks per lane and more (more variants unrolled: slower, instruction cache)
#define MINBLK 3               // resident blocks per SM the kernels are compiled for

template <int ORDER> struct PCQ { static constexpr int v = ORDER >= 4 ? 12 : (ORDER >= 2 ? 3 : 1); }; // float4 per staged cell

__device__ __forceinline__ float rsqrt_approx(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
    uint32_t s = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() {
    asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
}

// ---- fp32 lane arithmetic: scalar and packed pairs ------------------------------------------------
// Blackwell executes add/mul/fma on PAIRS of fp32 in one instruction (PTX *.f32x2 -> SASS FADD2, FMUL2,
// FFMA2): the same 128 lane-operations per SM per clock as the scalar forms, for half the issue
// slots.  The interaction kernels are issue-bound in scalar form, so every
// lane evaluates its sinks two at a time; an odd sink count leaves one scalar sink.
struct f2 { unsigned long long v; };
__device__ __forceinline__ f2 mk2(float lo, float hi) { f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ float lo2(f2 a) { float x; asm("{ .reg .f32 t; mov.b64 {%0, t}, %1; }" : "=f"(x) : "l"(a.v)); return x; }
__device__ __forceinline__ float hi2(f2 a) { float y; asm("{ .reg .f32 t; mov.b64 {t, %0}, %1; }" : "=f"(y) : "l"(a.v)); return y; }
__device__ __forceinline__ f2 operator+(f2 a, f2 b) { f2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
__device__ __forceinline__ f2 operator-(f2 a, f2 b) { f2 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
__device__ __forceinline__ f2 operator*(f2 a, f2 b) { f2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
__device__ __forceinline__ f2 vfma(f2 a, f2 b, f2 c) { f2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(a.v), "l"(b.v), "l"(c.v)); return r; }
__device__ __forceinline__ float vfma(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ f2 vrsqrt(f2 a) { return mk2(rsqrt_approx(lo2(a)), rsqrt_approx(hi2(a))); }
__device__ __forceinline__ float vrsqrt(float a) { return rsqrt_approx(a); }
template <class T> __device__ __forceinline__ T splat(float x);
template <> __device__ __forceinline__ float splat<float>(float x) { return x; }
template <> __device__ __forceinline__ f2 splat<f2>(float x) { return mk2(x, x); }

// ---- S8: one body on one sink (T = float) or on a pair of sinks (T = f2) --------------------------
// ns = NEGATED staged body (-x, -y, -z, -m) relative to the group origin; x = sink position(s).
// d = x - s;  a += (-m) ri^3 d;  phi += (-m) ri.   13 FP32-pipe operations + 1 MUFU.RSQ per sink.
template <class T>
__device__ __forceinline__ void pp_one(const float4 ns, const T (&x)[3], const float eps2, T (&a)[4]) {
    const T dx = x[0] + splat<T>(ns.x), dy = x[1] + splat<T>(ns.y), dz = x[2] + splat<T>(ns.z);
    const T r2 = vfma(dx, dx, vfma(dy, dy, vfma(dz, dz, splat<T>(eps2))));
    const T ri = vrsqrt(r2);
    const T ri2 = ri * ri, nmr = splat<T>(ns.w) * ri, nmr3 = nmr * ri2;
    a[0] = vfma(nmr3, dx, a[0]);
    a[1] = vfma(nmr3, dy, a[1]);
    a[2] = vfma(nmr3, dz, a[2]);
    a[3] = a[3] + nmr;
}
// the group's own bodies: the j = i slot is masked by index (works for eps = 0)
__device__ __forceinline__ void pp_one_self(const float4 ns, const bool same, const float (&x)[3], const float eps2, float (&a)[4]) {
    const float dx = x[0] + ns.x, dy = x[1] + ns.y, dz = x[2] + ns.z;
    const float r2 = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, eps2)));
    float ri = rsqrt_approx(r2);
    ri = same ? 0.0f : ri;
    const float ri2 = ri * ri, nmr = ns.w * ri, nmr3 = nmr * ri2;
    a[0] = fmaf(nmr3, dx, a[0]); a[1] = fmaf(nmr3, dy, a[1]); a[2] = fmaf(nmr3, dz, a[2]);
    a[3] += nmr;
}

// ---- f-4: cubic-spline softening (R-17) ------------------------------------------------
// A body is a ball of radius h = 2.8 eps with the spline density; with u = r / h the pair force m (s - x) fac and
// potential -m npot are  u <= 1/2: fac h^3 = 32/3 - 192/5 u^2 + 32 u^3,            npot h = 14/5 - 16/3 u^2 + 48/5 u^4 - 32/5 u^5
//                        u <= 1  : fac h^3 = 64/3 - 48u + 192/5 u^2 - 32/3 u^3 - 1/(15 u^3),
//                                  npot h = 16/5 - 1/(15u) - 32/3 u^2 + 16 u^3 - 48/5 u^4 + 32/15 u^5;   u > 1: Newtonian.
__device__ __forceinline__ void spline_kernel(const float r2, const float hinv, float& fac, float& npot) {
    const float ri = rsqrt_approx(fmaxf(r2, 1e-30f)), r = r2 * ri, u = r * hinv, u2 = u * u, hinv3 = hinv * hinv * hinv;
    const float fi = fmaf(u2, fmaf(32.0f, u, -38.4f), 10.6666667f);
    const float pi = fmaf(u2, fmaf(u2, fmaf(-6.4f, u, 9.6f), -5.33333333f), 2.8f);
    const float iu = __fdividef(1.0f, fmaxf(u, 0.25f)), iu3 = iu * iu * iu; // the middle branch is used for u >= 1/2 only
    const float fm = fmaf(u, fmaf(u, fmaf(-10.6666667f, u, 38.4f), -48.0f), 21.3333333f) - 0.0666666667f * iu3;
    const float pm = fmaf(u2, fmaf(u, fmaf(u, fmaf(2.13333333f, u, -9.6f), 16.0f), -10.6666667f), 3.2f) - 0.0666666667f * iu;
    const bool in = u < 0.5f, mid = u < 1.0f;
    fac = in ? hinv3 * fi : (mid ? hinv3 * fm : ri * ri * ri);
    npot = in ? hinv * pi : (mid ? hinv * pm : ri);
}
__device__ __forceinline__ void pp_one_spline(const float4 ns, const bool skip, const float (&x)[3], const float hinv, float (&a)[4]) {
    const float dx = x[0] + ns.x, dy = x[1] + ns.y, dz = x[2] + ns.z;
    float fac, npot;
    spline_kernel(fmaf(dx, dx, fmaf(dy, dy, dz * dz)), hinv, fac, npot);
    if (skip) { fac = 0.0f; npot = 0.0f; }
    const float nmf = ns.w * fac;
    a[0] = fmaf(nmf, dx, a[0]); a[1] = fmaf(nmf, dy, a[1]); a[2] = fmaf(nmf, dz, a[2]);
    a[3] = fmaf(ns.w, npot, a[3]);
}
__device__ __forceinline__ void pp_pair_spline(const float4 ns, const bool skip0, const bool skip1, const f2 (&x)[3], const float hinv, f2 (&a)[4]) {
    const f2 dx = x[0] + splat<f2>(ns.x), dy = x[1] + splat<f2>(ns.y), dz = x[2] + splat<f2>(ns.z);
    const f2 r2 = vfma(dx, dx, vfma(dy, dy, dz * dz));
    float f0, p0, f1, p1;
    spline_kernel(lo2(r2), hinv, f0, p0);
    spline_kernel(hi2(r2), hinv, f1, p1);
    if (skip0) { f0 = 0.0f; p0 = 0.0f; }
    if (skip1) { f1 = 0.0f; p1 = 0.0f; }
    const f2 nm = splat<f2>(ns.w), nmf = nm * mk2(f0, f1);
    a[0] = vfma(nmf, dx, a[0]); a[1] = vfma(nmf, dy, a[1]); a[2] = vfma(nmf, dz, a[2]);
    a[3] = vfma(nm, mk2(p0, p1), a[3]);
}

// ---- S9: one cell on one sink or a pair of sinks, eq (5) with g = (R^2+eps^2)^(-1/2) ----------------
// (DESIGN.md "P-C formulas").  R = x - z, D_k = (-1)^k (2k-1)!! u^-(2k+1)/2, raw moments, traces.
// Staged cell j of a batch: float4 slot q of the record sits at st[q*32 + j] (slot-major, so the
// K streams of a warp read K consecutive float4 -- no bank conflicts for any K):
//   slot 0: (-zx, -zy, -zz, -M0)  NEGATED centre of mass relative to the group origin, negated mass
//   slot 1: 3 (xx, xy, xz, yy)  slot 2: (3 yz, 3 zz, 1.5 t2, 0.5 t2)          ORDER >= 2  (the cellE2 record)
//   slots 3..11: M3 (10) M4 (15) t3 (3) T4 (6: xx xy xz yy yz zz) t4 (1) pad   ORDER >= 4
template <int ORDER, class T>
__device__ __forceinline__ void pc_one(const float4 q0, const float4 q1, const float4 q2, const float* __restrict__ m,
                                       const T (&x)[3], const float eps2, T (&a)[4]) {
    const T Rx = x[0] + splat<T>(q0.x), Ry = x[1] + splat<T>(q0.y), Rz = x[2] + splat<T>(q0.z);
    const T u = vfma(Rx, Rx, vfma(Ry, Ry, vfma(Rz, Rz, splat<T>(eps2))));
    const T ri = vrsqrt(u);
    const T ri2 = ri * ri, ri3 = ri * ri2;
    const T nm0 = splat<T>(q0.w);
    if (ORDER < 2) {
        const T c = nm0 * ri3;
        a[0] = vfma(c, Rx, a[0]); a[1] = vfma(c, Ry, a[1]); a[2] = vfma(c, Rz, a[2]);
        a[3] = vfma(nm0, ri, a[3]);
        return;
    }
    // quadrupole with the staged N = 3 M2, 1.5 t2 and 0.5 t2; ri5 = u^-5/2, w7 = -2.5 u^-1:
    //   phi = -M0 ri + 0.5 t2 ri3 - 0.5 ri5 (R N R);   a = R (-M0 ri3 + 1.5 t2 ri5 + w7 ri5 (R N R)) + ri5 (N R)
    const T ri5 = ri3 * ri2, w7 = splat<T>(-2.5f) * ri2;
    const T Mx = vfma(splat<T>(q1.x), Rx, vfma(splat<T>(q1.y), Ry, splat<T>(q1.z) * Rz));
    const T My = vfma(splat<T>(q1.y), Rx, vfma(splat<T>(q1.w), Ry, splat<T>(q2.x) * Rz));
    const T Mz = vfma(splat<T>(q1.z), Rx, vfma(splat<T>(q2.x), Ry, splat<T>(q2.y) * Rz));
    const T Q2 = vfma(Mx, Rx, vfma(My, Ry, Mz * Rz));
    const T hQ = ri5 * Q2;                                          // 3 u^-5/2 (R M2 R)
    T cR = vfma(hQ, w7, vfma(splat<T>(q2.z), ri5, nm0 * ri3));      // -7.5 u^-7/2 Q2 + 1.5 t2 u^-5/2 - M0 u^-3/2
    T ph = vfma(splat<T>(-0.5f), hQ, vfma(splat<T>(q2.w), ri3, nm0 * ri));
    const T D2 = ri5;                                               // multiplies N R = 3 M2 R
    if (ORDER < 4) { // accumulate straight into the partial sums
        a[0] = vfma(cR, Rx, vfma(D2, Mx, a[0]));
        a[1] = vfma(cR, Ry, vfma(D2, My, a[1]));
        a[2] = vfma(cR, Rz, vfma(D2, Mz, a[2]));
        a[3] = a[3] + ph;
        return;
    }
    T vx = D2 * Mx, vy = D2 * My, vz = D2 * Mz;
    {
        const T ri5 = ri3 * ri2, ri7 = ri5 * ri2, ri9 = ri7 * ri2, ri11 = ri9 * ri2;
        const T D2f = splat<T>(3.0f) * ri5, D3 = splat<T>(-15.0f) * ri7, D4 = splat<T>(105.0f) * ri9, D5 = splat<T>(-945.0f) * ri11;
        const float* m3 = m;          // 10
        const float* m4 = m + 10;     // 15
        const float* t3 = m + 25;     // 3
        const float* T4 = m + 28;     // 6: xx xy xz yy yz zz
        const T t4 = splat<T>(m[34]);
#define SP(v) splat<T>(v)
        const T xx = Rx * Rx, yy = Ry * Ry, zz = Rz * Rz, xy = Rx * Ry, xz = Rx * Rz, yz = Ry * Rz;
        const T xy2 = xy + xy, xz2 = xz + xz, yz2 = yz + yz;
        // V3_k = M3_ijk R_i R_j
        const T V3x = vfma(SP(m3[0]), xx, vfma(SP(m3[1]), xy2, vfma(SP(m3[2]), xz2, vfma(SP(m3[3]), yy, vfma(SP(m3[4]), yz2, SP(m3[5]) * zz)))));
        const T V3y = vfma(SP(m3[1]), xx, vfma(SP(m3[3]), xy2, vfma(SP(m3[4]), xz2, vfma(SP(m3[6]), yy, vfma(SP(m3[7]), yz2, SP(m3[8]) * zz)))));
        const T V3z = vfma(SP(m3[2]), xx, vfma(SP(m3[4]), xy2, vfma(SP(m3[5]), xz2, vfma(SP(m3[7]), yy, vfma(SP(m3[8]), yz2, SP(m3[9]) * zz)))));
        const T S3 = vfma(V3x, Rx, vfma(V3y, Ry, V3z * Rz));
        const T T3 = vfma(SP(t3[0]), Rx, vfma(SP(t3[1]), Ry, SP(t3[2]) * Rz));
        // cubic monomials with multiplicities: W4_k = M4_ijlk R_i R_j R_l
        const T c3 = SP(3.0f);
        const T cxxx = xx * Rx, cyyy = yy * Ry, czzz = zz * Rz;
        const T cxxy = c3 * xx * Ry, cxxz = c3 * xx * Rz, cxyy = c3 * Rx * yy, cxzz = c3 * Rx * zz;
        const T cyyz = c3 * yy * Rz, cyzz = c3 * Ry * zz, cxyz = SP(6.0f) * xy * Rz;
        const T W4x = vfma(SP(m4[0]), cxxx, vfma(SP(m4[1]), cxxy, vfma(SP(m4[2]), cxxz, vfma(SP(m4[3]), cxyy, vfma(SP(m4[4]), cxyz,
                      vfma(SP(m4[5]), cxzz, vfma(SP(m4[6]), cyyy, vfma(SP(m4[7]), cyyz, vfma(SP(m4[8]), cyzz, SP(m4[9]) * czzz)))))))));
        const T W4y = vfma(SP(m4[1]), cxxx, vfma(SP(m4[3]), cxxy, vfma(SP(m4[4]), cxxz, vfma(SP(m4[6]), cxyy, vfma(SP(m4[7]), cxyz,
                      vfma(SP(m4[8]), cxzz, vfma(SP(m4[10]), cyyy, vfma(SP(m4[11]), cyyz, vfma(SP(m4[12]), cyzz, SP(m4[13]) * czzz)))))))));
        const T W4z = vfma(SP(m4[2]), cxxx, vfma(SP(m4[4]), cxxy, vfma(SP(m4[5]), cxxz, vfma(SP(m4[7]), cxyy, vfma(SP(m4[8]), cxyz,
                      vfma(SP(m4[9]), cxzz, vfma(SP(m4[11]), cyyy, vfma(SP(m4[12]), cyyz, vfma(SP(m4[13]), cyzz, SP(m4[14]) * czzz)))))))));
        const T S4 = vfma(W4x, Rx, vfma(W4y, Ry, W4z * Rz));
        const T Ux = vfma(SP(T4[0]), Rx, vfma(SP(T4[1]), Ry, SP(T4[2]) * Rz));
        const T Uy = vfma(SP(T4[1]), Rx, vfma(SP(T4[3]), Ry, SP(T4[4]) * Rz));
        const T Uz = vfma(SP(T4[2]), Rx, vfma(SP(T4[4]), Ry, SP(T4[5]) * Rz));
        const T Q4 = vfma(Ux, Rx, vfma(Uy, Ry, Uz * Rz));
        // phi3 = (D3 S3 + 3 D2 T3)/6 ; phi4 = -(D4 S4 + 6 D3 Q4 + 3 D2 t4)/24
        ph = vfma(D3 * SP(1.0f / 6.0f), S3, vfma(SP(0.5f) * D2f, T3, ph));
        ph = vfma(D4 * SP(-1.0f / 24.0f), S4, vfma(SP(-0.25f) * D3, Q4, vfma(SP(-0.125f) * D2f, t4, ph)));
        // a3 = -[D4 S3 R + 3 D3 V3 + 3 D3 T3 R + 3 D2 t3]/6
        // a4 = [D5 S4 R + 4 D4 W4 + 6 D4 Q4 R + 12 D3 U + 3 D3 t4 R]/24
        cR = vfma(D4 * SP(-1.0f / 6.0f), S3, vfma(SP(-0.5f) * D3, T3, cR));
        cR = vfma(D5 * SP(1.0f / 24.0f), S4, vfma(SP(0.25f) * D4, Q4, vfma(SP(0.125f) * D3, t4, cR)));
        const T hD3n = SP(-0.5f) * D3, hD2n = SP(-0.5f) * D2f, sD4 = D4 * SP(1.0f / 6.0f), hD3p = SP(0.5f) * D3;
        vx = vfma(hD3n, V3x, vfma(hD2n, SP(t3[0]), vfma(sD4, W4x, vfma(hD3p, Ux, vx))));
        vy = vfma(hD3n, V3y, vfma(hD2n, SP(t3[1]), vfma(sD4, W4y, vfma(hD3p, Uy, vy))));
        vz = vfma(hD3n, V3z, vfma(hD2n, SP(t3[2]), vfma(sD4, W4z, vfma(hD3p, Uz, vz))));
#undef SP
    }
    a[0] = a[0] + vfma(cR, Rx, vx);
    a[1] = a[1] + vfma(cR, Ry, vy);
    a[2] = a[2] + vfma(cR, Rz, vz);
    a[3] = a[3] + ph;
}

// ---- the sinks of one lane: NP pairs + (S odd) one scalar ------------------------------------------
template <int S> struct Sinks {
    static constexpr int NP = S / 2, TAIL = S & 1;
    f2 x2[NP ? NP : 1][3], a2[NP ? NP : 1][4];
    float x1[3], a1[4];
    int me[S];
    __device__ __forceinline__ void zero_partials() {
#pragma unroll
        for (int p = 0; p < NP; ++p)
#pragma unroll
            for (int k = 0; k < 4; ++k) a2[p][k] = mk2(0.f, 0.f);
#pragma unroll
        for (int k = 0; k < 4; ++k) a1[k] = 0.f;
    }
    __device__ __forceinline__ void set_x(int i, float vx, float vy, float vz) { // slot i (compile-time after unrolling)
        if (TAIL && i == S - 1) { x1[0] = vx; x1[1] = vy; x1[2] = vz; return; }
        const int p = i >> 1;
        if (i & 1) { x2[p][0] = mk2(lo2(x2[p][0]), vx); x2[p][1] = mk2(lo2(x2[p][1]), vy); x2[p][2] = mk2(lo2(x2[p][2]), vz); }
        else { x2[p][0] = mk2(vx, 0.f); x2[p][1] = mk2(vy, 0.f); x2[p][2] = mk2(vz, 0.f); }
    }
    __device__ __forceinline__ float get_a(int i, int k) const {
        if (TAIL && i == S - 1) return a1[k];
        return (i & 1) ? hi2(a2[i >> 1][k]) : lo2(a2[i >> 1][k]);
    }
    __device__ __forceinline__ void pp(const float4 ns, float eps2) {
#pragma unroll
        for (int p = 0; p < NP; ++p) pp_one<f2>(ns, x2[p], eps2, a2[p]);
        if (TAIL) pp_one<float>(ns, x1, eps2, a1);
    }
    // the group's own bodies: the same packed arithmetic, the j = i slot masked by index through ri = 0 (works for eps = 0)
    __device__ __forceinline__ void pp_self(const float4 ns, int j, float eps2) {
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            const f2 dx = x2[p][0] + splat<f2>(ns.x), dy = x2[p][1] + splat<f2>(ns.y), dz = x2[p][2] + splat<f2>(ns.z);
            const f2 r2 = vfma(dx, dx, vfma(dy, dy, vfma(dz, dz, splat<f2>(eps2))));
            const float r0 = rsqrt_approx(lo2(r2)), r1 = rsqrt_approx(hi2(r2));
            const f2 ri = mk2(j == me[2 * p] ? 0.0f : r0, j == me[2 * p + 1] ? 0.0f : r1);
            const f2 ri2 = ri * ri, nmr = splat<f2>(ns.w) * ri, nmr3 = nmr * ri2;
            a2[p][0] = vfma(nmr3, dx, a2[p][0]); a2[p][1] = vfma(nmr3, dy, a2[p][1]); a2[p][2] = vfma(nmr3, dz, a2[p][2]);
            a2[p][3] = a2[p][3] + nmr;
        }
        if (TAIL) pp_one_self(ns, j == me[S - 1], x1, eps2, a1);
    }
    __device__ __forceinline__ void pp_spline(const float4 ns, int j, float hinv) { // j: index in the group if ns is one of its own bodies, else -1 (me[] >= 0 or -1 for idle slots: an idle slot never equals j >= 0... nor -1 matters: its result is dropped)
#pragma unroll
        for (int p = 0; p < NP; ++p) pp_pair_spline(ns, j >= 0 && j == me[2 * p], j >= 0 && j == me[2 * p + 1], x2[p], hinv, a2[p]);
        if (TAIL) pp_one_spline(ns, j >= 0 && j == me[S - 1], x1, hinv, a1);
    }
    template <int ORDER>
    __device__ __forceinline__ void pc(const float4 q0, const float4 q1, const float4 q2, const float* m, float eps2) {
#pragma unroll
        for (int p = 0; p < NP; ++p) pc_one<ORDER, f2>(q0, q1, q2, m, x2[p], eps2, a2[p]);
        if (TAIL) pc_one<ORDER, float>(q0, q1, q2, m, x1, eps2, a1);
    }
};

// ---- per-warp shared-memory layout (byte offsets from the warp's base) -------------------------
template <int ORDER> struct WL {
    static constexpr int NQ = PCQ<ORDER>::v;
    static constexpr int pcst = 0;                               // 2 x [NQ][32] float4  staged cells
    static constexpr int ppst = pcst + 2 * NQ * 32 * 16;         // 2 x [32] float4      staged bodies
    static constexpr int accum = ppst + 2 * 32 * 16;             // [SMAX*4][32] double  running sums (acc, pot) per lane
    static constexpr int bytes = accum + SMAX * 4 * 32 * 8;
};

// ---- S8/S9/S10: one chunk (<= 32*SMAX sinks) of one group -----------------------------------------
// L = 1 << lgL lanes per source stream, S = ceil(nchunk / L) sinks per lane.
template <int ORDER, bool PER, int S, bool SPL>
__device__ __noinline__ void eval_chunk(const ForceArgs& P, const int w, const GroupRec g, const int64_t gi, const uint32_t chunk0,
                                        const uint32_t nchunk, const int lgL, const int lane) {
    using Lay = WL<ORDER>;
    constexpr int NQ = Lay::NQ;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    unsigned char* const base = smem_raw + (size_t)w * Lay::bytes;
    float4* const pcst = reinterpret_cast<float4*>(base + Lay::pcst);
    float4* const ppst = reinterpret_cast<float4*>(base + Lay::ppst);
    double* const As = reinterpret_cast<double*>(base + Lay::accum) + lane; // this lane's running sums: As[(4 i + k) * 32]

    const int L = 1 << lgL, lgK = 5 - lgL, K = 1 << lgK; // lanes per stream, source streams
    const int sl = lane & (L - 1);                       // lane inside its stream
    const int strm = lane >> lgL;                        // stream id: takes sources strm, strm + K, ...
    // origin of the relative coordinates: fp32-rounded centre of the group cube
    double ox, oy, oz;
    {
        const WalkCell gw = P.wcell[g.cell];
        const int gs = 1 << (HOT_MAXLEVEL - (int)(gw.w >> 27));
        const int gox = (int)(gw.x & 0x1fffffu), goy = (int)((gw.x >> 21) | ((gw.y & 0x3ffu) << 11)), goz = (int)((gw.y >> 10) & 0x1fffffu);
        const double h = P.size * (1.0 / 2097152.0);
        ox = (double)(float)(P.lo[0] + ((double)gox + 0.5 * gs) * h);
        oy = (double)(float)(P.lo[1] + ((double)goy + 0.5 * gs) * h);
        oz = (double)(float)(P.lo[2] + ((double)goz + 0.5 * gs) * h);
    }
    // sinks: slot i of lane sl holds body chunk0 + i*L + sl of the group (every stream holds them all)
    Sinks<S> sk;
#pragma unroll
    for (int i = 0; i < S; ++i) {
        const uint32_t loc = (uint32_t)(i * L + sl);
        sk.me[i] = loc < nchunk ? (int)(chunk0 + loc) : -1;
        const float4 b = P.body[g.first + (loc < nchunk ? chunk0 + loc : 0u)];
        sk.set_x(i, (float)((double)b.x - ox), (float)((double)b.y - oy), (float)((double)b.z - oz));
#pragma unroll
        for (int k = 0; k < 4; ++k) As[(4 * i + k) * 32] = 0.0;
    }
    sk.zero_partials();
    const float eps2 = SPL ? 0.0f : P.eps2; // spline softening: accepted cells lie beyond its support, their expansions are Newtonian
    const float hinv = P.hinv;
    // fp32 partials are added to the fp64 running sums after at most ~32 sources per lane
    int nacc = 0;
    auto flush = [&]() {
#pragma unroll
        for (int i = 0; i < S; ++i)
#pragma unroll
            for (int k = 0; k < 4; ++k) As[(4 * i + k) * 32] += (double)sk.get_a(i, k);
        sk.zero_partials();
        nacc = 0;
    };
    auto shift_of = [&](int im, double& shx, double& shy, double& shz) {
        shx = (double)(im / 25 - 2) * P.size; shy = (double)((im / 5) % 5 - 2) * P.size; shz = (double)(im % 5 - 2) * P.size;
    };
    // sources are staged NEGATED (origin - position, -mass): the kernels then need no negations

    // ---- the group's own bodies (the "self block"): the walk leaves the group cell out ----------
    for (uint32_t j0 = 0; j0 < (P.do_pp ? g.count : 0u); j0 += BATCH) {
        const int cnt = (int)min((uint32_t)BATCH, g.count - j0);
        if (lane < cnt) {
            const float4 b = P.body[g.first + j0 + lane];
            ppst[lane] = make_float4((float)(ox - (double)b.x), (float)(oy - (double)b.y), (float)(oz - (double)b.z), -b.w);
        }
        __syncwarp();
#pragma unroll 1
        for (int j = strm; j < cnt; j += K) { if (SPL) sk.pp_spline(ppst[j], (int)j0 + j, hinv); else sk.pp_self(ppst[j], (int)j0 + j, eps2); }
        __syncwarp();
    }
    flush();

    // ---- S9: the particle-cell list ------------------------------------------------------------------
    {
        unsigned long long o0 = P.pcoff[gi];
        int n = (int)P.lpc[gi];
        if (P.seg >= 0) { // tolerance mode: the list is monopoles | quadrupoles | hexadecapoles, this launch takes one part
            const int n0 = (int)P.lpc0[gi], n2 = (int)P.lpc2[gi];
            if (P.seg == 0) n = n0;
            else if (P.seg == 1) { o0 += n0; n = n2; }
            else { o0 += n0 + n2; n -= n0 + n2; }
        }
        const uint32_t* const pl = P.pclist + o0;
        const uint8_t* const pi = PER ? P.pcimg + o0 : nullptr;
        const int nb = (n + BATCH - 1) / BATCH;
        CellA cA;
        cA.zx = cA.zy = cA.zz = 0.0; cA.m0 = 0.f; cA.bmax = 0.f;
        uint32_t cnext = 0; int inext = 62, pim = 62;
        auto fetch_idx = [&](int b) { // list entries of batch b
            if (b * BATCH + lane < n) { cnext = pl[b * BATCH + lane]; if (PER) inext = pi[b * BATCH + lane]; }
        };
        auto issue = [&](int b) { // gather batch b: centre to registers, moments straight to shared memory
            if (b * BATCH + lane < n) {
                const uint32_t c = PER ? (cnext & ~HOT_COARSE_FLAG) : cnext;
                pim = inext;
                cA = P.cellA[c];
                if (PER && (cnext & HOT_COARSE_FLAG)) cA.m0 = 0.f; // its monopole is summed in fp64 elsewhere (hot_periodic.cu)
                float4* const dst = pcst + (b & 1) * NQ * BATCH + lane;
                if (ORDER >= 2) {
                    const float4* src = reinterpret_cast<const float4*>(P.cellE2 + c);
                    cp_async16(dst + 1 * BATCH, src);
                    cp_async16(dst + 2 * BATCH, src + 1);
                }
                if (ORDER >= 4) {
                    const float4* src = reinterpret_cast<const float4*>(P.cellM34 + c);
#pragma unroll
                    for (int k = 0; k < 9; ++k) cp_async16(dst + (3 + k) * BATCH, src + k);
                }
            }
        };
        if (nb > 0) { fetch_idx(0); issue(0); fetch_idx(1); }
        for (int b = 0; b < nb; ++b) {
            const int cnt = min(BATCH, n - b * BATCH);
            float4* const st = pcst + (b & 1) * NQ * BATCH;
            if (lane < cnt) {
                double shx = 0, shy = 0, shz = 0;
                if (PER) shift_of(pim, shx, shy, shz);
                st[lane] = make_float4((float)(ox - (cA.zx + shx)), (float)(oy - (cA.zy + shy)), (float)(oz - (cA.zz + shz)), -cA.m0);
            }
            if (ORDER >= 2) cp_async_wait_all();
            __syncwarp();
            if (b + 1 < nb) { issue(b + 1); fetch_idx(b + 2); } // in flight during the arithmetic below
            if (ORDER < 4) { // the next source's record is read while the current one is evaluated
                int j = strm;
                float4 n0 = st[j < cnt ? j : 0], n1 = n0, n2 = n0;
                if (ORDER >= 2) { n1 = st[32 + (j < cnt ? j : 0)]; n2 = st[64 + (j < cnt ? j : 0)]; }
                if (S >= UNROLL2_S) { // two sources per trip: the sums stay in their registers (no copies at the loop end)
#pragma unroll 2
                while (j < cnt) {
                    const float4 q0 = n0, q1 = n1, q2 = n2;
                    j += K;
                    const int jn = j < cnt ? j : strm;
                    n0 = st[jn];
                    if (ORDER >= 2) { n1 = st[32 + jn]; n2 = st[64 + jn]; }
                    sk.template pc<ORDER>(q0, q1, q2, nullptr, eps2);
                }
                } else {
#pragma unroll 1
                while (j < cnt) {
                    const float4 q0 = n0, q1 = n1, q2 = n2;
                    j += K;
                    const int jn = j < cnt ? j : strm;
                    n0 = st[jn];
                    if (ORDER >= 2) { n1 = st[32 + jn]; n2 = st[64 + jn]; }
                    sk.template pc<ORDER>(q0, q1, q2, nullptr, eps2);
                }
                }
            } else {
#pragma unroll 1
                for (int j = strm; j < cnt; j += K) {
                    const float4 q0 = st[j], q1 = st[32 + j], q2 = st[64 + j];
                    float m[36];
#pragma unroll
                    for (int k = 0; k < 9; ++k) {
                        const float4 t = st[(3 + k) * 32 + j];
                        m[4 * k] = t.x; m[4 * k + 1] = t.y; m[4 * k + 2] = t.z; m[4 * k + 3] = t.w;
                    }
                    sk.template pc<ORDER>(q0, q1, q2, m, eps2);
                }
            }
            nacc += (cnt + K - 1) >> lgK;
            if (nacc >= FLUSH_N) flush();
        }
        __syncwarp();
    }
    // ---- S8: the particle-particle list ------------------------------------------------------------
    {
        const unsigned long long o0 = P.ppoff[gi];
        const int n = P.do_pp ? (int)P.lpp[gi] : 0;
        const uint32_t* const pl = P.pplist + o0;
        const uint8_t* const pi = PER ? P.ppimg + o0 : nullptr;
        const int nb = (n + BATCH - 1) / BATCH;
        float4 pb = make_float4(0.f, 0.f, 0.f, 0.f);
        uint32_t cnext = 0; int inext = 62, pim = 62;
        auto fetch_idx = [&](int b) {
            if (b * BATCH + lane < n) { cnext = pl[b * BATCH + lane]; if (PER) inext = pi[b * BATCH + lane]; }
        };
        auto issue = [&](int b) {
            if (b * BATCH + lane < n) { pb = P.body[cnext]; pim = inext; }
        };
        if (nb > 0) { fetch_idx(0); issue(0); fetch_idx(1); }
        for (int b = 0; b < nb; ++b) {
            const int cnt = min(BATCH, n - b * BATCH);
            float4* const st = ppst + (b & 1) * BATCH;
            if (lane < cnt) {
                double shx = 0, shy = 0, shz = 0;
                if (PER) shift_of(pim, shx, shy, shz);
                st[lane] = make_float4((float)(ox - ((double)pb.x + shx)), (float)(oy - ((double)pb.y + shy)),
                                       (float)(oz - ((double)pb.z + shz)), -pb.w);
            }
            __syncwarp();
            if (b + 1 < nb) { issue(b + 1); fetch_idx(b + 2); }
            {
                int j = strm;
                float4 nx = st[j < cnt ? j : 0];
#pragma unroll 2
                while (j < cnt) {
                    const float4 sb = nx;
                    j += K;
                    nx = st[j < cnt ? j : strm];
                    if (SPL) sk.pp_spline(sb, -1, hinv); else sk.pp(sb, eps2);
                }
            }
            nacc += (cnt + K - 1) >> lgK;
            if (nacc >= FLUSH_N) flush();
        }
        __syncwarp();
    }
    flush();
    // combine the K streams' partial sums
    double A[S][4];
#pragma unroll
    for (int i = 0; i < S; ++i)
#pragma unroll
        for (int k = 0; k < 4; ++k) A[i][k] = As[(4 * i + k) * 32];
    for (int off = L; off < 32; off <<= 1) {
#pragma unroll
        for (int i = 0; i < S; ++i)
#pragma unroll
            for (int k = 0; k < 4; ++k) A[i][k] += __shfl_xor_sync(FULL, A[i][k], off);
    }
    // S10: results to the caller's particle order (periodic: plus the far field, still in fp64)
    if (strm == 0) {
#pragma unroll
        for (int i = 0; i < S; ++i) {
            if (sk.me[i] >= 0) {
                const uint32_t o = P.perm[g.first + sk.me[i]];
                if (PER && P.far) {
                    const double4 f = reinterpret_cast<const double4*>(P.far)[g.first + sk.me[i]];
                    A[i][0] += f.x; A[i][1] += f.y; A[i][2] += f.z; A[i][3] += f.w;
                }
                if (P.accumulate) { // a later launch of the same hot_forces call (tolerance mode: one launch per order)
                    A[i][0] += (double)P.acc[3 * (int64_t)o]; A[i][1] += (double)P.acc[3 * (int64_t)o + 1]; A[i][2] += (double)P.acc[3 * (int64_t)o + 2];
                    if (P.pot) A[i][3] += (double)P.pot[o];
                }
                P.acc[3 * (int64_t)o] = (float)A[i][0];
                P.acc[3 * (int64_t)o + 1] = (float)A[i][1];
                P.acc[3 * (int64_t)o + 2] = (float)A[i][2];
                if (P.pot) P.pot[o] = (float)A[i][3];
            }
        }
    }
}

// one pass over the group's lists for sinks [c0, c0 + nc) with L = 1 << lgL lanes per source stream
template <int ORDER, bool PER, bool SPL>
__device__ __forceinline__ void run_chunk(const ForceArgs& P, const int w, const GroupRec g, const int64_t gi, const uint32_t c0,
                                          const uint32_t nc, const int lgL, const int lane) {
    const int S = (int)((nc + (1u << lgL) - 1) >> lgL);
    if (S <= 1) eval_chunk<ORDER, PER, 1, SPL>(P, w, g, gi, c0, nc, lgL, lane);
    else if (S == 2) eval_chunk<ORDER, PER, 2, SPL>(P, w, g, gi, c0, nc, lgL, lane);
    else if (S == 3) eval_chunk<ORDER, PER, 3, SPL>(P, w, g, gi, c0, nc, lgL, lane);
    else if (S == 4) eval_chunk<ORDER, PER, 4, SPL>(P, w, g, gi, c0, nc, lgL, lane);
    else if (S == 5) eval_chunk<ORDER, PER, 5, SPL>(P, w, g, gi, c0, nc, lgL, lane);
    else eval_chunk<ORDER, PER, 6, SPL>(P, w, g, gi, c0, nc, lgL, lane);
    static_assert(SMAX == 6, "one eval_chunk instance per sinks-per-lane count");
}
// smallest stream width that holds n sinks with at most SMAX per lane
__device__ __forceinline__ int fit_lgL(uint32_t n) {
    int lgL = 0;
    while (((n + (1u << lgL) - 1) >> lgL) > SMAX) ++lgL;
    return lgL;
}
// Relative time of a pass: L lanes per stream each spend (PLAN_A + PLAN_B * S) per source, 32 / L sources at a time;
// PLAN_C is what a pass costs whatever its sinks (list reads, staging of the sources).
#define PLAN_A 1
#define PLAN_B 3
#define PLAN_C 12
__device__ __forceinline__ int pass_cost(int lgL, uint32_t n) { return (PLAN_A + PLAN_B * (int)((n + (1u << lgL) - 1) >> lgL)) << lgL; }

// The passes of one group.  Sinks in passes of at most 32*SMAX (full passes first: 6 sinks per lane is the most
// efficient blocking, measured against an even split).  The last nc sinks: one pass with ceil(nc / L) sinks per lane
// leaves up to L - 1 of its slots idle; when cheaper, a pass with floor(nc / L) full slots per lane is followed by a
// narrow pass for the < L sinks left over (e.g. 100 sinks: 32 x 3 + 4 x 1 instead of 32 x 4).
template <class F>
__device__ __forceinline__ void plan_group(const uint32_t count, F&& emit) {
    for (uint32_t c0 = 0; c0 < count; c0 += 32 * SMAX) {
        const uint32_t nc = min((uint32_t)(32 * SMAX), count - c0);
        int lgL = fit_lgL(nc);
        uint32_t nmain = nc;
        int best = pass_cost(lgL, nc);
#pragma unroll 1
        for (int lg = 0; lg <= 5; ++lg) {
            const uint32_t sf = nc >> lg;
            if (sf < 1 || sf > SMAX) continue;
            const uint32_t r = nc - (sf << lg);
            if (r == 0) continue; // an exact fit is the single pass already
            const int c = pass_cost(lg, sf << lg) + pass_cost(fit_lgL(r), r) + PLAN_C;
            if (c < best) { best = c; lgL = lg; nmain = sf << lg; }
        }
        emit(c0, nmain, lgL);
        if (nmain < nc) emit(c0 + nmain, nc - nmain, fit_lgL(nc - nmain));
    }
}
#ifndef HOT_FORCES_PERIODIC_TU
// Work items of the interaction kernel, one per pass: (group - g0, first sink, sinks, lg2 lanes per stream).  The SMAX
// variants of the loops together do not fit the instruction cache (unrolling all of them: 76 -> 105 ms), so the items are
// ordered by sinks per lane, 6 first -- but only INSIDE superblocks of 2^sb_shift consecutive groups (key order), so that
// the groups in flight at any time are neighbours in space and share the cells and bodies of their lists in L2.
// cls: [nsb][8] items per (superblock, class = SMAX - sinks per lane), [nsb][8] where each starts, [nsb][8] fill cursors,
// [1] total.  FILL = false counts, plan_scan_kernel places the classes, FILL = true fills.
template <bool FILL>
__global__ void __launch_bounds__(256) plan_kernel(const __grid_constant__ ForceArgs P) {
    __shared__ unsigned int s_cnt[8], s_base[8];
    if (threadIdx.x < 8) s_cnt[threadIdx.x] = 0;
    __syncthreads();
    const int64_t gi = P.g0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned int sb = (unsigned int)(((int64_t)blockIdx.x * blockDim.x) >> P.sb_shift); // sb_shift >= 8: one superblock per block
    const uint32_t count = gi < P.g1 ? P.group[gi].count : 0u;
    plan_group(count, [&](uint32_t, uint32_t nc, int lgL) { atomicAdd(&s_cnt[SMAX - (int)((nc + (1u << lgL) - 1) >> lgL)], 1u); });
    __syncthreads();
    if (!FILL) {
        if (threadIdx.x < 8 && s_cnt[threadIdx.x]) atomicAdd(&P.cls[8 * sb + threadIdx.x], s_cnt[threadIdx.x]);
        return;
    }
    if (threadIdx.x < 8) { // the block's range in every class: start of the class + a cursor
        s_base[threadIdx.x] = P.cls[8 * (P.nsb + sb) + threadIdx.x] + (s_cnt[threadIdx.x] ? atomicAdd(&P.cls[8 * (2 * P.nsb + sb) + threadIdx.x], s_cnt[threadIdx.x]) : 0u);
        s_cnt[threadIdx.x] = 0;
    }
    __syncthreads();
    plan_group(count, [&](uint32_t c0, uint32_t nc, int lgL) {
        const int c = SMAX - (int)((nc + (1u << lgL) - 1) >> lgL);
        P.items[s_base[c] + atomicAdd(&s_cnt[c], 1u)] = make_uint4((uint32_t)(gi - P.g0), c0, nc, (uint32_t)lgL);
    });
}
// exclusive scan of the 8 nsb (superblock, class) counts in that order; one warp
__global__ void __launch_bounds__(32) plan_scan_kernel(unsigned int* __restrict__ cls, unsigned int nsb) {
    const int lane = threadIdx.x;
    unsigned int carry = 0;
    for (unsigned int b = 0; b < 8 * nsb; b += 32) {
        const unsigned int v = b + lane < 8 * nsb ? cls[b + lane] : 0u;
        unsigned int x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const unsigned int y = __shfl_up_sync(FULL, x, o); if (lane >= o) x += y; }
        if (b + lane < 8 * nsb) cls[8 * nsb + b + lane] = carry + x - v;
        carry += __shfl_sync(FULL, x, 31);
    }
    if (lane == 0) cls[24 * nsb] = carry;
}
size_t plan_cls_elems(int64_t ng, int sb_shift) { return 24 * (size_t)((ng + ((int64_t)1 << sb_shift) - 1) >> sb_shift) + 1; }
cudaError_t launch_plan(const ForceArgs& a, cudaStream_t st) {
    const int64_t ng = a.g1 - a.g0;
    if (ng <= 0) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(a.cls, 0, plan_cls_elems(ng, a.sb_shift) * sizeof(unsigned int), st);
    if (e != cudaSuccess) return e;
    HOT_LAUNCHED(3);
    plan_kernel<false><<<(unsigned)((ng + 255) / 256), 256, 0, st>>>(a);
    plan_scan_kernel<<<1, 32, 0, st>>>(a.cls, a.nsb);
    plan_kernel<true><<<(unsigned)((ng + 255) / 256), 256, 0, st>>>(a);
    return cudaGetLastError();
}
#endif

template <int ORDER, bool PER, bool SPL>
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32, ORDER >= 4 ? 3 : MINBLK) forces_kernel(const __grid_constant__ ForceArgs P) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const unsigned int total = P.cls[24 * P.nsb];
    while (true) {
        unsigned int q = 0;
        if (lane == 0) q = atomicAdd(P.counter, 1u);
        q = __shfl_sync(FULL, q, 0);
        if (q >= total) break;
        const uint4 it = P.items[q];
        const int64_t gi = P.g0 + (int64_t)it.x;
        run_chunk<ORDER, PER, SPL>(P, w, P.group[gi], gi, it.y, it.z, (int)it.w, lane);
    }
}

template <int ORDER, bool PER, bool SPL> static cudaError_t launch_one(const ForceArgs& a, cudaStream_t st) {
    constexpr int smem = WL<ORDER>::bytes * WARPS_PER_BLOCK;
    static int nblocks = 0;
    if (!nblocks) {
        cudaError_t e = cudaFuncSetAttribute(forces_kernel<ORDER, PER, SPL>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        int dev = 0, nsm = 0, occ = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, forces_kernel<ORDER, PER, SPL>, WARPS_PER_BLOCK * 32, smem);
        if (e != cudaSuccess) return e;
        nblocks = nsm * (occ < 1 ? 1 : occ);
    }
    HOT_LAUNCHED(1);
    forces_kernel<ORDER, PER, SPL><<<nblocks, WARPS_PER_BLOCK * 32, smem, st>>>(a);
    return cudaGetLastError();
}
#ifndef HOT_FORCES_PERIODIC_TU
cudaError_t dispatch_periodic(const ForceArgs& a, cudaStream_t st);
cudaError_t launch_forces(const ForceArgs& a, cudaStream_t st) {
    if (a.periodic) return dispatch_periodic(a, st);
    if (a.spline) {
        if (a.order >= 4) return launch_one<4, false, true>(a, st);
        if (a.order >= 2) return launch_one<2, false, true>(a, st);
        return launch_one<0, false, true>(a, st);
    }
    if (a.order >= 4) return launch_one<4, false, false>(a, st);
    if (a.order >= 2) return launch_one<2, false, false>(a, st);
    return launch_one<0, false, false>(a, st);
}
#else
cudaError_t dispatch_periodic(const ForceArgs& a, cudaStream_t st) {
    if (a.spline) {
        if (a.order >= 4) return launch_one<4, true, true>(a, st);
        if (a.order >= 2) return launch_one<2, true, true>(a, st);
        return launch_one<0, true, true>(a, st);
    }
    if (a.order >= 4) return launch_one<4, true, false>(a, st);
    if (a.order >= 2) return launch_one<2, true, false>(a, st);
    return launch_one<0, true, false>(a, st);
}
#endif

// hot_interact.cuh -- the fp32 interaction arithmetic shared by the evaluation kernels (hot_forces.cu, hot_bg.cu):
// packed-pair helpers, S8 particle-particle, cubic-spline kernel, S9 particle-cell of eq (5) through order 4.
#pragma once
#include "hot_internal.h"

__device__ __forceinline__ float rsqrt_approx(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
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
// DIP (background-subtracted cells, expanded about the cell centre: hot_bg.cu, R-18): qd = (M1x, M1y, M1z, -) adds
//   phi_1 = D1 (M1 . R) = -ri^3 (M1 . R),   a_1 = -[D2 (M1 . R) R + D1 M1] = -3 ri^5 (M1 . R) R + ri^3 M1.
template <int ORDER, class T, bool DIP = false>
__device__ __forceinline__ void pc_one(const float4 q0, const float4 q1, const float4 q2, const float* __restrict__ m,
                                       const T (&x)[3], const float eps2, T (&a)[4], const float4 qd = make_float4(0.f, 0.f, 0.f, 0.f)) {
    const T Rx = x[0] + splat<T>(q0.x), Ry = x[1] + splat<T>(q0.y), Rz = x[2] + splat<T>(q0.z);
    const T u = vfma(Rx, Rx, vfma(Ry, Ry, vfma(Rz, Rz, splat<T>(eps2))));
    const T ri = vrsqrt(u);
    const T ri2 = ri * ri, ri3 = ri * ri2;
    const T nm0 = splat<T>(q0.w);
    if (ORDER < 2) {
        T c = nm0 * ri3;
        if (DIP) {
            const T dR = vfma(splat<T>(qd.x), Rx, vfma(splat<T>(qd.y), Ry, splat<T>(qd.z) * Rz)), w = ri3 * dR;
            c = vfma(splat<T>(-3.0f) * ri2, w, c);
            a[0] = vfma(ri3, splat<T>(qd.x), a[0]); a[1] = vfma(ri3, splat<T>(qd.y), a[1]); a[2] = vfma(ri3, splat<T>(qd.z), a[2]);
            a[3] = a[3] - w;
        }
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
    if (DIP) {
        const T dR = vfma(splat<T>(qd.x), Rx, vfma(splat<T>(qd.y), Ry, splat<T>(qd.z) * Rz));
        cR = vfma(splat<T>(-3.0f) * ri5, dR, cR);
        ph = ph - ri3 * dR;
        a[0] = vfma(ri3, splat<T>(qd.x), a[0]); a[1] = vfma(ri3, splat<T>(qd.y), a[1]); a[2] = vfma(ri3, splat<T>(qd.z), a[2]);
    }
    const T D2 = ri5;                                               // multiplies N R = 3 M2 R
    if (ORDER < 4) { // accumulate straight into the partial sums
        a[0] = vfma(cR, Rx, vfma(D2, Mx, a[0]));
        a[1] = vfma(cR, Ry, vfma(D2, My, a[1]));
        a[2] = vfma(cR, Rz, vfma(D2, Mz, a[2]));
        a[3] = a[3] + ph;
        return;
    }
    T vx = D2 * Mx, vy = D2 * My, vz = D2 * Mz;
    T cP; // coefficient of P = R / u in the acceleration (degrees 3 and 4)
    T Px, Py, Pz;
    {
        // Degrees 3 and 4 in P = R u^-1 instead of R: every contraction of an n-th moment with k copies of R carries u^-k with it, so
        // the coefficients left are ri, ri3 and ri5 only.  With R itself they are ri7 ... ri11, and ri11 overflows fp32 for
        // |R| < 5.8e-4 length units although the term it multiplies is tiny there -- the error-bound criterion accepts small
        // cells that close (inf accelerations at N >= 2^22 in tolerance mode before this), an opening angle at level >= 12.
        //   S3 = M3 PPP, V3 = M3 PP, T3 = t3 P, S4 = M4 PPPP, W4 = M4 PPP, Q4 = T4 PP, U = T4 P;
        //   phi3 = (-15 ri S3 + 9 ri3 T3)/6          phi4 = -(105 ri S4 - 90 ri3 Q4 + 9 ri5 t4)/24
        //   a3 = -[105 ri S3 P - 45 ri3 V3 - 45 ri3 T3 P + 9 ri5 t3]/6
        //   a4 = [-945 ri S4 P + 420 ri3 W4 + 630 ri3 Q4 P - 180 ri5 U - 45 ri5 t4 P]/24
        Px = Rx * ri2; Py = Ry * ri2; Pz = Rz * ri2;
        const float* m3 = m;          // 10
        const float* m4 = m + 10;     // 15
        const float* t3 = m + 25;     // 3
        const float* T4 = m + 28;     // 6: xx xy xz yy yz zz
        const T t4 = splat<T>(m[34]);
#define SP(v) splat<T>(v)
        const T xx = Px * Px, yy = Py * Py, zz = Pz * Pz, xy = Px * Py, xz = Px * Pz, yz = Py * Pz;
        const T xy2 = xy + xy, xz2 = xz + xz, yz2 = yz + yz;
        // V3_k = M3_ijk P_i P_j
        const T V3x = vfma(SP(m3[0]), xx, vfma(SP(m3[1]), xy2, vfma(SP(m3[2]), xz2, vfma(SP(m3[3]), yy, vfma(SP(m3[4]), yz2, SP(m3[5]) * zz)))));
        const T V3y = vfma(SP(m3[1]), xx, vfma(SP(m3[3]), xy2, vfma(SP(m3[4]), xz2, vfma(SP(m3[6]), yy, vfma(SP(m3[7]), yz2, SP(m3[8]) * zz)))));
        const T V3z = vfma(SP(m3[2]), xx, vfma(SP(m3[4]), xy2, vfma(SP(m3[5]), xz2, vfma(SP(m3[7]), yy, vfma(SP(m3[8]), yz2, SP(m3[9]) * zz)))));
        const T S3 = vfma(V3x, Px, vfma(V3y, Py, V3z * Pz));
        const T T3 = vfma(SP(t3[0]), Px, vfma(SP(t3[1]), Py, SP(t3[2]) * Pz));
        // cubic monomials with multiplicities: W4_k = M4_ijlk P_i P_j P_l
        const T c3 = SP(3.0f);
        const T cxxx = xx * Px, cyyy = yy * Py, czzz = zz * Pz;
        const T cxxy = c3 * xx * Py, cxxz = c3 * xx * Pz, cxyy = c3 * Px * yy, cxzz = c3 * Px * zz;
        const T cyyz = c3 * yy * Pz, cyzz = c3 * Py * zz, cxyz = SP(6.0f) * xy * Pz;
        const T W4x = vfma(SP(m4[0]), cxxx, vfma(SP(m4[1]), cxxy, vfma(SP(m4[2]), cxxz, vfma(SP(m4[3]), cxyy, vfma(SP(m4[4]), cxyz,
                      vfma(SP(m4[5]), cxzz, vfma(SP(m4[6]), cyyy, vfma(SP(m4[7]), cyyz, vfma(SP(m4[8]), cyzz, SP(m4[9]) * czzz)))))))));
        const T W4y = vfma(SP(m4[1]), cxxx, vfma(SP(m4[3]), cxxy, vfma(SP(m4[4]), cxxz, vfma(SP(m4[6]), cxyy, vfma(SP(m4[7]), cxyz,
                      vfma(SP(m4[8]), cxzz, vfma(SP(m4[10]), cyyy, vfma(SP(m4[11]), cyyz, vfma(SP(m4[12]), cyzz, SP(m4[13]) * czzz)))))))));
        const T W4z = vfma(SP(m4[2]), cxxx, vfma(SP(m4[4]), cxxy, vfma(SP(m4[5]), cxxz, vfma(SP(m4[7]), cxyy, vfma(SP(m4[8]), cxyz,
                      vfma(SP(m4[9]), cxzz, vfma(SP(m4[11]), cyyy, vfma(SP(m4[12]), cyyz, vfma(SP(m4[13]), cyzz, SP(m4[14]) * czzz)))))))));
        const T S4 = vfma(W4x, Px, vfma(W4y, Py, W4z * Pz));
        const T Ux = vfma(SP(T4[0]), Px, vfma(SP(T4[1]), Py, SP(T4[2]) * Pz));
        const T Uy = vfma(SP(T4[1]), Px, vfma(SP(T4[3]), Py, SP(T4[4]) * Pz));
        const T Uz = vfma(SP(T4[2]), Px, vfma(SP(T4[4]), Py, SP(T4[5]) * Pz));
        const T Q4 = vfma(Ux, Px, vfma(Uy, Py, Uz * Pz));
        const T r1a = SP(-2.5f) * ri, r1b = SP(-4.375f) * ri, r3a = SP(1.5f) * ri3, r3b = SP(3.75f) * ri3, r5a = SP(-0.375f) * ri5;
        ph = vfma(r1a, S3, vfma(r3a, T3, ph));                               // -15/6 ri S3 + 9/6 ri3 T3
        ph = vfma(r1b, S4, vfma(r3b, Q4, vfma(r5a, t4, ph)));                // -105/24 ri S4 + 90/24 ri3 Q4 - 9/24 ri5 t4
        const T r1c = SP(-17.5f) * ri, r3c = SP(7.5f) * ri3, r1d = SP(-39.375f) * ri, r3d = SP(26.25f) * ri3, r5d = SP(-1.875f) * ri5;
        cP = vfma(r1c, S3, r3c * T3);                                        // -105/6 ri S3 + 45/6 ri3 T3
        cP = vfma(r1d, S4, vfma(r3d, Q4, vfma(r5d, t4, cP)));                // -945/24 ri S4 + 630/24 ri3 Q4 - 45/24 ri5 t4
        const T r5e = SP(-1.5f) * ri5, r3e = SP(17.5f) * ri3, r5f = SP(-7.5f) * ri5;
        vx = vfma(r3c, V3x, vfma(r5e, SP(t3[0]), vfma(r3e, W4x, vfma(r5f, Ux, vx)))); // 45/6 ri3 V3 - 9/6 ri5 t3 + 420/24 ri3 W4 - 180/24 ri5 U
        vy = vfma(r3c, V3y, vfma(r5e, SP(t3[1]), vfma(r3e, W4y, vfma(r5f, Uy, vy))));
        vz = vfma(r3c, V3z, vfma(r5e, SP(t3[2]), vfma(r3e, W4z, vfma(r5f, Uz, vz))));
#undef SP
    }
    a[0] = a[0] + vfma(cR, Rx, vfma(cP, Px, vx));
    a[1] = a[1] + vfma(cR, Ry, vfma(cP, Py, vy));
    a[2] = a[2] + vfma(cR, Rz, vfma(cP, Pz, vz));
    a[3] = a[3] + ph;
}


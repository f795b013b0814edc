// hot_forces.cu -- S7 walk fused with S8 particle-particle and S9 particle-cell kernels, S10 scatter.
//
// One warp owns one sink group at a time (persistent grid, dynamic group counter).  The warp walks
// the tree cooperatively: it pops up to 32 cells from a shared-memory stack, every lane applies
// the multipole acceptance criterion to one cell (integer geometry, one IEEE double multiply and
// compare -- DESIGN.md R-7), and ballots sort the cells into
//   accepted  -> cell index appended to the particle-cell list (shared memory),
//   rejected leaf -> its bodies staged into the particle-particle list (shared memory),
//   else      -> its children pushed on the stack.
// Whenever a list holds a batch of 32 sources the warp evaluates it: sources are read from shared
// memory as broadcast 128-bit loads, the sinks (S per lane, S = ceil(n_G/32)) live in registers
// (the m x n blocking of PAPER.md:162-164).  The lists are never written to HBM.
//
// Arithmetic: interactions in fp32 (FFMA + MUFU.RSQ), coordinates relative to the group centre
// (formed in fp64 when a source is staged), batch partial sums in fp32, running sums in fp64.
#include "hot_internal.h"

#define FULL 0xffffffffu
#define STACK_CAP 512          // per-warp traversal stack in shared memory (entries)
#define BATCH 32               // sources per evaluation batch
#define WARPS_PER_BLOCK 4

__device__ __forceinline__ float rsqrt_approx(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <int ORDER> struct PCQ { static constexpr int v = ORDER >= 4 ? 12 : (ORDER >= 2 ? 3 : 1); }; // float4 per staged cell

// ---- S8: one body on S sinks ------------------------------------------------------------------
// 3 FADD + 3 FFMA + MUFU.RSQ + 3 FMUL + 3 FFMA + 1 FADD per sink: 13 FP32-pipe instructions + 1 MUFU
template <int S>
__device__ __forceinline__ void pp_eval(const float4 s, const float (&x)[S][3], float eps2, float (&a)[S][4]) {
#pragma unroll
    for (int i = 0; i < S; ++i) {
        float dx = s.x - x[i][0], dy = s.y - x[i][1], dz = s.z - x[i][2];
        float r2 = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, eps2)));
        float ri = rsqrt_approx(r2);
        float ri2 = ri * ri, mr = s.w * ri, mr3 = mr * ri2;
        a[i][0] = fmaf(mr3, dx, a[i][0]);
        a[i][1] = fmaf(mr3, dy, a[i][1]);
        a[i][2] = fmaf(mr3, dz, a[i][2]);
        a[i][3] -= mr;
    }
}
// the group's own bodies: the j = i slot is masked by index (works for eps = 0)
template <int S>
__device__ __forceinline__ void pp_eval_self(const float4 s, int j, const int (&me)[S], const float (&x)[S][3], float eps2,
                                             float (&a)[S][4]) {
#pragma unroll
    for (int i = 0; i < S; ++i) {
        float dx = s.x - x[i][0], dy = s.y - x[i][1], dz = s.z - x[i][2];
        float r2 = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, eps2)));
        float ri = rsqrt_approx(r2);
        ri = (j == me[i]) ? 0.0f : ri;
        float ri2 = ri * ri, mr = s.w * ri, mr3 = mr * ri2;
        a[i][0] = fmaf(mr3, dx, a[i][0]);
        a[i][1] = fmaf(mr3, dy, a[i][1]);
        a[i][2] = fmaf(mr3, dz, a[i][2]);
        a[i][3] -= mr;
    }
}

// ---- S9: one cell on S sinks, eq (5) with g = (R^2+eps^2)^(-1/2) ------
// R = x - z, D_k = (-1)^k (2k-1)!! u^-(2k+1)/2, raw moments, traces t2, t3, T4, t4.
template <int ORDER, int S>
__device__ __forceinline__ void pc_eval(const float4* __restrict__ q, const float (&x)[S][3], float eps2, float (&a)[S][4]) {
    const float4 q0 = q[0];
    float4 q1, q2;
    if (ORDER >= 2) { q1 = q[1]; q2 = q[2]; }
#pragma unroll
    for (int i = 0; i < S; ++i) {
        const float Rx = x[i][0] - q0.x, Ry = x[i][1] - q0.y, Rz = x[i][2] - q0.z;
        const float u = fmaf(Rx, Rx, fmaf(Ry, Ry, fmaf(Rz, Rz, eps2)));
        const float ri = rsqrt_approx(u);
        const float ri2 = ri * ri, ri3 = ri * ri2;
        if (ORDER < 2) {
            const float c = -q0.w * ri3;
            a[i][0] = fmaf(c, Rx, a[i][0]); a[i][1] = fmaf(c, Ry, a[i][1]); a[i][2] = fmaf(c, Rz, a[i][2]);
            a[i][3] = fmaf(-q0.w, ri, a[i][3]);
            continue;
        }
        const float ri5 = ri3 * ri2, ri7 = ri5 * ri2;
        // quadrupole: M2 = (xx xy xz yy | yz zz t2)
        const float Mx = fmaf(q1.x, Rx, fmaf(q1.y, Ry, q1.z * Rz));
        const float My = fmaf(q1.y, Rx, fmaf(q1.w, Ry, q2.x * Rz));
        const float Mz = fmaf(q1.z, Rx, fmaf(q2.x, Ry, q2.y * Rz));
        const float Q2 = fmaf(Mx, Rx, fmaf(My, Ry, Mz * Rz));
        const float t2 = q2.z;
        const float D2 = 3.0f * ri5, hD3 = -7.5f * ri7; // D2, D3/2
        // coefficient of R and potential through order 2
        float cR = fmaf(hD3, Q2, fmaf(0.5f * D2, t2, -q0.w * ri3));
        float ph = fmaf(0.5f * ri3, t2, fmaf(-0.5f * D2, Q2, -q0.w * ri));
        float vx = D2 * Mx, vy = D2 * My, vz = D2 * Mz;
        if (ORDER >= 4) {
            const float ri9 = ri7 * ri2, ri11 = ri9 * ri2;
            const float D3 = -15.0f * ri7, D4 = 105.0f * ri9, D5 = -945.0f * ri11;
            const float* m3 = reinterpret_cast<const float*>(q + 3);      // 10
            const float* m4 = m3 + 10;                                    // 15
            const float* t3 = m3 + 25;                                    // 3
            const float* T4 = m3 + 28;                                    // 6: xx xy xz yy yz zz
            const float t4 = m3[34];
            const float xx = Rx * Rx, yy = Ry * Ry, zz = Rz * Rz, xy = Rx * Ry, xz = Rx * Rz, yz = Ry * Rz;
            const float xy2 = xy + xy, xz2 = xz + xz, yz2 = yz + yz;
            // V3_k = M3_ijk R_i R_j
            const float V3x = fmaf(m3[0], xx, fmaf(m3[1], xy2, fmaf(m3[2], xz2, fmaf(m3[3], yy, fmaf(m3[4], yz2, m3[5] * zz)))));
            const float V3y = fmaf(m3[1], xx, fmaf(m3[3], xy2, fmaf(m3[4], xz2, fmaf(m3[6], yy, fmaf(m3[7], yz2, m3[8] * zz)))));
            const float V3z = fmaf(m3[2], xx, fmaf(m3[4], xy2, fmaf(m3[5], xz2, fmaf(m3[7], yy, fmaf(m3[8], yz2, m3[9] * zz)))));
            const float S3 = fmaf(V3x, Rx, fmaf(V3y, Ry, V3z * Rz));
            const float T3 = fmaf(t3[0], Rx, fmaf(t3[1], Ry, t3[2] * Rz));
            // cubic monomials with multiplicities: W4_k = M4_ijlk R_i R_j R_l
            const float cxxx = xx * Rx, cyyy = yy * Ry, czzz = zz * Rz;
            const float cxxy = 3.0f * xx * Ry, cxxz = 3.0f * xx * Rz, cxyy = 3.0f * Rx * yy, cxzz = 3.0f * Rx * zz;
            const float cyyz = 3.0f * yy * Rz, cyzz = 3.0f * Ry * zz, cxyz = 6.0f * xy * Rz;
            const float W4x = fmaf(m4[0], cxxx, fmaf(m4[1], cxxy, fmaf(m4[2], cxxz, fmaf(m4[3], cxyy, fmaf(m4[4], cxyz,
                              fmaf(m4[5], cxzz, fmaf(m4[6], cyyy, fmaf(m4[7], cyyz, fmaf(m4[8], cyzz, m4[9] * czzz)))))))));
            const float W4y = fmaf(m4[1], cxxx, fmaf(m4[3], cxxy, fmaf(m4[4], cxxz, fmaf(m4[6], cxyy, fmaf(m4[7], cxyz,
                              fmaf(m4[8], cxzz, fmaf(m4[10], cyyy, fmaf(m4[11], cyyz, fmaf(m4[12], cyzz, m4[13] * czzz)))))))));
            const float W4z = fmaf(m4[2], cxxx, fmaf(m4[4], cxxy, fmaf(m4[5], cxxz, fmaf(m4[7], cxyy, fmaf(m4[8], cxyz,
                              fmaf(m4[9], cxzz, fmaf(m4[11], cyyy, fmaf(m4[12], cyyz, fmaf(m4[13], cyzz, m4[14] * czzz)))))))));
            const float S4 = fmaf(W4x, Rx, fmaf(W4y, Ry, W4z * Rz));
            const float Ux = fmaf(T4[0], Rx, fmaf(T4[1], Ry, T4[2] * Rz));
            const float Uy = fmaf(T4[1], Rx, fmaf(T4[3], Ry, T4[4] * Rz));
            const float Uz = fmaf(T4[2], Rx, fmaf(T4[4], Ry, T4[5] * Rz));
            const float Q4 = fmaf(Ux, Rx, fmaf(Uy, Ry, Uz * Rz));
            // phi3 = (D3 S3 + 3 D2 T3)/6 ; phi4 = -(D4 S4 + 6 D3 Q4 + 3 D2 t4)/24
            ph = fmaf(D3 * (1.0f / 6.0f), S3, fmaf(0.5f * D2, T3, ph));
            ph = fmaf(-D4 * (1.0f / 24.0f), S4, fmaf(-0.25f * D3, Q4, fmaf(-0.125f * D2, t4, ph)));
            // a3 = -[D4 S3 R + 3 D3 V3 + 3 D3 T3 R + 3 D2 t3]/6
            // a4 = [D5 S4 R + 4 D4 W4 + 6 D4 Q4 R + 12 D3 U + 3 D3 t4 R]/24
            cR = fmaf(-D4 * (1.0f / 6.0f), S3, fmaf(-0.5f * D3, T3, cR));
            cR = fmaf(D5 * (1.0f / 24.0f), S4, fmaf(0.25f * D4, Q4, fmaf(0.125f * D3, t4, cR)));
            const float hD3n = -0.5f * D3, hD2n = -0.5f * D2, sD4 = D4 * (1.0f / 6.0f), hD3p = 0.5f * D3;
            vx = fmaf(hD3n, V3x, fmaf(hD2n, t3[0], fmaf(sD4, W4x, fmaf(hD3p, Ux, vx))));
            vy = fmaf(hD3n, V3y, fmaf(hD2n, t3[1], fmaf(sD4, W4y, fmaf(hD3p, Uy, vy))));
            vz = fmaf(hD3n, V3z, fmaf(hD2n, t3[2], fmaf(sD4, W4z, fmaf(hD3p, Uz, vz))));
        }
        a[i][0] += fmaf(cR, Rx, vx);
        a[i][1] += fmaf(cR, Ry, vy);
        a[i][2] += fmaf(cR, Rz, vz);
        a[i][3] += ph;
    }
}

struct WarpSmem {
    uint32_t* stack;   // [STACK_CAP]
    uint32_t* pcidx;   // [2*BATCH]
    float4* ppbuf;     // [2*BATCH]
    float4* pcbuf;     // [BATCH * PCQ]
    uint8_t* stimg;    // [STACK_CAP]  (periodic) image id per stack entry
    uint8_t* pcimg;    // [2*BATCH]
};
template <int ORDER, bool PER> __host__ __device__ constexpr int warp_smem_bytes() {
    return STACK_CAP * 4 + 2 * BATCH * 4 + 2 * BATCH * 16 + BATCH * PCQ<ORDER>::v * 16 + (PER ? STACK_CAP + 2 * BATCH : 0);
}

// fp32 batch partials -> fp64 running sums
template <int S> __device__ __forceinline__ void flush_acc(float (&a)[S][4], double (&A)[S][4]) {
#pragma unroll
    for (int i = 0; i < S; ++i)
#pragma unroll
        for (int k = 0; k < 4; ++k) { A[i][k] += (double)a[i][k]; a[i][k] = 0.0f; }
}

template <int ORDER, bool PER, int S>
__device__ __noinline__ void process_chunk(const ForceArgs& P, const WarpSmem& sm, const GroupRec g, uint32_t chunk0, uint32_t nchunk,
                                           bool first_chunk, uint32_t* gstack, int lane, unsigned long long& nvisit,
                                           unsigned long long& nspill, uint64_t& Lpc, uint64_t& Lpp) {
    constexpr int NQ = PCQ<ORDER>::v;
    const uint32_t lt = (1u << lane) - 1u;
    // group cube on the integer grid
    const WalkCell gw = P.wcell[g.cell];
    const int glev = (int)(gw.w >> 27);
    const int gs = 1 << (HOT_MAXLEVEL - glev);
    const int gox = (int)(gw.x & 0x1fffffu), goy = (int)((gw.x >> 21) | ((gw.y & 0x3ffu) << 11)), goz = (int)((gw.y >> 10) & 0x1fffffu);
    // origin of the relative coordinates: fp32-rounded centre of the group cube
    const double h = P.size * (1.0 / 2097152.0);
    const float ocx = (float)(P.lo[0] + ((double)gox + 0.5 * gs) * h), ocy = (float)(P.lo[1] + ((double)goy + 0.5 * gs) * h),
                ocz = (float)(P.lo[2] + ((double)goz + 0.5 * gs) * h);
    const double ox = ocx, oy = ocy, oz = ocz;
    // sinks
    float x[S][3];
    int me[S];
    float a[S][4];
    double A[S][4];
#pragma unroll
    for (int i = 0; i < S; ++i) {
        uint32_t loc = chunk0 + i * 32 + lane;
        me[i] = loc < g.count ? (int)loc : -1;
        float4 b = P.body[g.first + (loc < g.count ? loc : 0)];
        x[i][0] = (float)((double)b.x - ox); x[i][1] = (float)((double)b.y - oy); x[i][2] = (float)((double)b.z - oz);
#pragma unroll
        for (int k = 0; k < 4; ++k) { a[i][k] = 0.0f; A[i][k] = 0.0; }
    }
    (void)nchunk;
    const float eps2 = P.eps2;
    int npc = 0, npp = 0; // pending list lengths

    auto eval_pp = [&](int cnt) {
#pragma unroll 4
        for (int k = 0; k < cnt; ++k) pp_eval<S>(sm.ppbuf[k], x, eps2, a);
        flush_acc<S>(a, A);
    };
    // stage `cnt` accepted cells (indices in pcidx[0..cnt)) and evaluate them
    auto eval_pc = [&](int cnt) {
        if (lane < cnt) {
            uint32_t c = sm.pcidx[lane];
            double shx = 0, shy = 0, shz = 0;
            if (PER) {
                int im = sm.pcimg[lane];
                shx = (double)(im / 25 - 2) * P.size; shy = (double)((im / 5) % 5 - 2) * P.size; shz = (double)(im % 5 - 2) * P.size;
            }
            const CellA cA = P.cellA[c];
            float4* dst = sm.pcbuf + lane * NQ;
            dst[0] = make_float4((float)(cA.zx + shx - ox), (float)(cA.zy + shy - oy), (float)(cA.zz + shz - oz), cA.m0);
            if (ORDER >= 2) {
                const float4* src = reinterpret_cast<const float4*>(P.cellM2 + c);
                float4 m0 = src[0], m1 = src[1];
                dst[1] = m0;
                dst[2] = make_float4(m1.x, m1.y, cA.t2, 0.0f);
            }
            if (ORDER >= 4) {
                const float4* src = reinterpret_cast<const float4*>(P.cellM34 + c);
#pragma unroll
                for (int k = 0; k < 9; ++k) dst[3 + k] = src[k];
            }
        }
        __syncwarp();
#pragma unroll 2
        for (int k = 0; k < cnt; ++k) pc_eval<ORDER, S>(sm.pcbuf + k * NQ, x, eps2, a);
        flush_acc<S>(a, A);
        __syncwarp();
    };

    // the group's own bodies (the "self block"): the walk skips the group cell itself
    for (uint32_t j0 = 0; j0 < g.count; j0 += BATCH) {
        uint32_t cnt = min((uint32_t)BATCH, g.count - j0);
        if (lane < cnt) {
            float4 b = P.body[g.first + j0 + lane];
            sm.ppbuf[lane] = make_float4((float)((double)b.x - ox), (float)((double)b.y - oy), (float)((double)b.z - oz), b.w);
        }
        __syncwarp();
        for (uint32_t k = 0; k < cnt; ++k) pp_eval_self<S>(sm.ppbuf[k], (int)(j0 + k), me, x, eps2, a);
        __syncwarp();
    }
    flush_acc<S>(a, A);
    if (first_chunk) Lpp += g.count;

    // traversal
    int top = 0, gtop = 0; // shared-memory stack height, spilled entries in the global arena
    const int nimg = PER ? 125 : 1;
    for (int img0 = 0; img0 < nimg; img0 += 32) {
        // seed: the root for each image (lane = image)
        {
            int im = img0 + lane;
            bool v = im < nimg;
            uint32_t m = __ballot_sync(FULL, v);
            if (v) { sm.stack[top + lane] = 0u; if (PER) sm.stimg[top + lane] = (uint8_t)(PER ? im : 0); }
            top += __popc(m);
            __syncwarp();
        }
        while (top > 0) {
            const int nt = min(top, 32);
            const bool v = lane < nt;
            uint32_t c = 0; int im = PER ? 62 : 0;
            if (v) { c = sm.stack[top - 1 - lane]; if (PER) im = sm.stimg[top - 1 - lane]; }
            top -= nt;
            __syncwarp();
            WalkCell wc = {0, 0, 0, 0};
            if (v) wc = P.wcell[c];
            nvisit += nt;
            const int lev = (int)(wc.w >> 27);
            const uint32_t cnt = wc.w & 0x7ffffffu;
            const bool leaf = (wc.y >> 31) != 0;
            int cx = (int)(wc.x & 0x1fffffu), cy = (int)((wc.x >> 21) | ((wc.y & 0x3ffu) << 11)), cz = (int)((wc.y >> 10) & 0x1fffffu);
            if (PER) { cx += (im / 25 - 2) << HOT_MAXLEVEL; cy += ((im / 5) % 5 - 2) << HOT_MAXLEVEL; cz += (im % 5 - 2) << HOT_MAXLEVEL; }
            const int s = 1 << (HOT_MAXLEVEL - lev);
            const int gx = max(0, max(cx - (gox + gs), gox - (cx + s)));
            const int gy = max(0, max(cy - (goy + gs), goy - (cy + s)));
            const int gz = max(0, max(cz - (goz + gs), goz - (cz + s)));
            const unsigned long long d2 = (unsigned long long)((long long)gx * gx) + (unsigned long long)((long long)gy * gy) +
                                          (unsigned long long)((long long)gz * gz);
            const double s2 = __longlong_as_double((long long)(1023 + 2 * (HOT_MAXLEVEL - lev)) << 52); // (double)(s*s), exact
            const bool acc = v && (s2 < P.theta2 * __ull2double_rn(d2));
            const bool self = v && c == g.cell && (!PER || im == 62);
            const bool rej_leaf = v && !acc && leaf && !self;
            const bool open = v && !acc && !leaf && !self;
            // accepted cells -> P-C list
            {
                uint32_t m = __ballot_sync(FULL, acc);
                if (acc) { int p = npc + __popc(m & lt); sm.pcidx[p] = c; if (PER) sm.pcimg[p] = (uint8_t)im; }
                int na = __popc(m);
                npc += na;
                if (first_chunk) Lpc += na;
                __syncwarp();
                if (npc >= BATCH) {
                    eval_pc(BATCH);
                    npc -= BATCH;
                    if (lane < npc) { // move the remainder down
                        uint32_t t = sm.pcidx[BATCH + lane]; uint8_t ti = PER ? sm.pcimg[BATCH + lane] : 0;
                        sm.pcidx[lane] = t; if (PER) sm.pcimg[lane] = ti;
                    }
                    __syncwarp();
                }
            }
            // rejected leaves -> stage their bodies into the P-P list
            {
                uint32_t m = __ballot_sync(FULL, rej_leaf);
                while (m) {
                    const int src = __ffs(m) - 1;
                    m &= m - 1;
                    const uint32_t f = __shfl_sync(FULL, wc.z, src), n = __shfl_sync(FULL, cnt, src);
                    double shx = 0, shy = 0, shz = 0;
                    if (PER) {
                        int si = __shfl_sync(FULL, im, src);
                        shx = (double)(si / 25 - 2) * P.size; shy = (double)((si / 5) % 5 - 2) * P.size; shz = (double)(si % 5 - 2) * P.size;
                    }
                    if (first_chunk) Lpp += n;
                    for (uint32_t j0 = 0; j0 < n; j0 += BATCH) {
                        const uint32_t k = min((uint32_t)BATCH, n - j0);
                        if ((uint32_t)lane < k) {
                            float4 b = P.body[f + j0 + lane];
                            sm.ppbuf[npp + lane] = make_float4((float)((double)b.x + shx - ox), (float)((double)b.y + shy - oy),
                                                               (float)((double)b.z + shz - oz), b.w);
                        }
                        npp += (int)k;
                        __syncwarp();
                        if (npp >= BATCH) {
                            eval_pp(BATCH);
                            npp -= BATCH;
                            __syncwarp();
                            if (lane < npp) { float4 t = sm.ppbuf[BATCH + lane]; sm.ppbuf[lane] = t; }
                            __syncwarp();
                        }
                    }
                }
            }
            // opened cells -> push children
            {
                uint32_t m = __ballot_sync(FULL, open);
                if (m) {
                    int nch = open ? (int)cnt : 0, pre = nch;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(FULL, pre, o); if (lane >= o) pre += y; }
                    const int total = __shfl_sync(FULL, pre, 31);
                    if (top + total > STACK_CAP) { // spill the bottom of the stack to the global arena
                        const int keep = top > 128 ? 128 : top, mv = top - keep; // keep a few on chip
                        if ((int64_t)gtop + mv > P.gstack_cap) { if (lane == 0) atomicOr(P.errflag, 4); top = 0; gtop = 0; break; }
                        for (int t = lane; t < mv; t += 32) {
                            gstack[gtop + t] = sm.stack[t];
                            if (PER) gstack[P.gstack_cap + gtop + t] = sm.stimg[t]; // image ids: second half of the arena
                        }
                        __syncwarp();
                        for (int t0 = 0; t0 < keep; t0 += 32) { // move the kept top down (ascending order is safe)
                            uint32_t e = 0; uint8_t ei = 0;
                            if (t0 + lane < keep) { e = sm.stack[mv + t0 + lane]; if (PER) ei = sm.stimg[mv + t0 + lane]; }
                            __syncwarp();
                            if (t0 + lane < keep) { sm.stack[t0 + lane] = e; if (PER) sm.stimg[t0 + lane] = ei; }
                            __syncwarp();
                        }
                        gtop += mv; top = keep; ++nspill;
                    }
                    if (open) {
                        int p = top + pre - nch;
                        for (int k = 0; k < nch; ++k) { sm.stack[p + k] = wc.z + k; if (PER) sm.stimg[p + k] = (uint8_t)im; }
                    }
                    top += total;
                    __syncwarp();
                }
            }
            if (top == 0 && gtop > 0) { // refill from the global arena
                const int mv = gtop > STACK_CAP / 2 ? STACK_CAP / 2 : gtop;
                for (int t = lane; t < mv; t += 32) {
                    sm.stack[t] = gstack[gtop - mv + t];
                    if (PER) sm.stimg[t] = (uint8_t)gstack[P.gstack_cap + gtop - mv + t];
                }
                gtop -= mv; top = mv;
                __syncwarp();
            }
        }
    }
    if (npc > 0) eval_pc(npc);
    if (npp > 0) eval_pp(npp);
    // S10: results to the caller's particle order
#pragma unroll
    for (int i = 0; i < S; ++i) {
        if (me[i] >= 0) {
            uint32_t o = P.perm[g.first + me[i]];
            P.acc[3 * (int64_t)o] = (float)A[i][0];
            P.acc[3 * (int64_t)o + 1] = (float)A[i][1];
            P.acc[3 * (int64_t)o + 2] = (float)A[i][2];
            if (P.pot) P.pot[o] = (float)A[i][3];
        }
    }
}

// SCAP = largest number of sinks per lane this instantiation can hold (ceil(NCRIT/32) rounded up to
// 2, 4 or 8); the register allocation of the kernel is that of its largest process_chunk.
template <int ORDER, bool PER, int SCAP>
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32) forces_kernel(const ForceArgs P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    constexpr int WB = warp_smem_bytes<ORDER, PER>();
    unsigned char* base = smem_raw + (size_t)w * WB;
    WarpSmem sm;
    sm.pcbuf = reinterpret_cast<float4*>(base);
    sm.ppbuf = sm.pcbuf + BATCH * PCQ<ORDER>::v;
    sm.stack = reinterpret_cast<uint32_t*>(sm.ppbuf + 2 * BATCH);
    sm.pcidx = sm.stack + STACK_CAP;
    sm.stimg = reinterpret_cast<uint8_t*>(sm.pcidx + 2 * BATCH);
    sm.pcimg = sm.stimg + STACK_CAP;
    const int64_t gwarp = (int64_t)blockIdx.x * WARPS_PER_BLOCK + w;
    uint32_t* gstack = P.gstack + gwarp * P.gstack_cap * (PER ? 2 : 1);
    unsigned long long nvisit = 0, nspill = 0, sum_pp = 0, sum_pc = 0;
    while (true) {
        unsigned int gi = 0;
        if (lane == 0) gi = atomicAdd(P.counter, 1u);
        gi = __shfl_sync(FULL, gi, 0);
        if ((int64_t)gi >= P.ngroups) break;
        const GroupRec g = P.group[gi];
        uint64_t Lpc = 0, Lpp = 0;
        // sinks in chunks of at most 32*SCAP (only finest-level groups can exceed one chunk)
        for (uint32_t c0 = 0; c0 < g.count; c0 += 32 * SCAP) {
            const uint32_t nc = min((uint32_t)(32 * SCAP), g.count - c0);
            const int S = (int)((nc + 31) / 32);
            const bool fc = c0 == 0;
            if (S <= 1) process_chunk<ORDER, PER, 1>(P, sm, g, c0, nc, fc, gstack, lane, nvisit, nspill, Lpc, Lpp);
            else if (S <= 2) process_chunk<ORDER, PER, 2>(P, sm, g, c0, nc, fc, gstack, lane, nvisit, nspill, Lpc, Lpp);
            else if (SCAP >= 4 && S <= 3) process_chunk<ORDER, PER, SCAP >= 4 ? 3 : 1>(P, sm, g, c0, nc, fc, gstack, lane, nvisit, nspill, Lpc, Lpp);
            else if (SCAP >= 4 && S <= 4) process_chunk<ORDER, PER, SCAP >= 4 ? 4 : 1>(P, sm, g, c0, nc, fc, gstack, lane, nvisit, nspill, Lpc, Lpp);
            else if (SCAP >= 8 && S <= 6) process_chunk<ORDER, PER, SCAP >= 8 ? 6 : 1>(P, sm, g, c0, nc, fc, gstack, lane, nvisit, nspill, Lpc, Lpp);
            else if (SCAP >= 8) process_chunk<ORDER, PER, SCAP >= 8 ? 8 : 1>(P, sm, g, c0, nc, fc, gstack, lane, nvisit, nspill, Lpc, Lpp);
        }
        if (lane == 0) {
            P.glpc[gi] = Lpc; P.glpp[gi] = Lpp;
            sum_pp += (unsigned long long)g.count * Lpp; sum_pc += (unsigned long long)g.count * Lpc;
        }
    }
    if (lane == 0) {
        atomicAdd(&P.stat[0], nvisit); atomicAdd(&P.stat[1], nspill);
        atomicAdd(&P.stat[2], sum_pp); atomicAdd(&P.stat[3], sum_pc);
    }
}

template <int ORDER, bool PER, int SCAP> static cudaError_t launch_one(const ForceArgs& a, int nblocks, cudaStream_t st, int* occ_out) {
    constexpr int WB = warp_smem_bytes<ORDER, PER>();
    const int smem = WB * WARPS_PER_BLOCK;
    cudaError_t e = cudaFuncSetAttribute(forces_kernel<ORDER, PER, SCAP>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    if (occ_out) {
        int occ = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, forces_kernel<ORDER, PER, SCAP>, WARPS_PER_BLOCK * 32, smem);
        *occ_out = occ;
        return e;
    }
    HOT_LAUNCHED(1);
    forces_kernel<ORDER, PER, SCAP><<<nblocks, WARPS_PER_BLOCK * 32, smem, st>>>(a);
    return cudaGetLastError();
}
template <int ORDER, bool PER> static cudaError_t launch_scap(const ForceArgs& a, int scap, int nblocks, cudaStream_t st, int* occ) {
    if (scap <= 2) return launch_one<ORDER, PER, 2>(a, nblocks, st, occ);
    if (scap <= 4) return launch_one<ORDER, PER, 4>(a, nblocks, st, occ);
    return launch_one<ORDER, PER, 8>(a, nblocks, st, occ);
}
#ifndef HOT_FORCES_PERIODIC_TU
cudaError_t dispatch_open(const ForceArgs& a, int nblocks, cudaStream_t st, int* occ) {
    if (a.order >= 4) return launch_scap<4, false>(a, a.scap, nblocks, st, occ);
    if (a.order >= 2) return launch_scap<2, false>(a, a.scap, nblocks, st, occ);
    return launch_scap<0, false>(a, a.scap, nblocks, st, occ);
}
cudaError_t dispatch_periodic(const ForceArgs& a, int nblocks, cudaStream_t st, int* occ);
static int g_num_sms = 0;
static int blocks_for(const ForceArgs& a) {
    if (!g_num_sms) {
        int dev = 0; cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&g_num_sms, cudaDevAttrMultiProcessorCount, dev);
    }
    int occ = 0;
    cudaError_t e = a.periodic ? dispatch_periodic(a, 0, nullptr, &occ) : dispatch_open(a, 0, nullptr, &occ);
    if (e != cudaSuccess || occ < 1) occ = 1;
    return g_num_sms * occ;
}
int force_grid_warps(int order, int periodic, int scap) {
    ForceArgs a{}; a.order = order; a.periodic = periodic; a.scap = scap;
    return blocks_for(a) * WARPS_PER_BLOCK;
}
cudaError_t launch_forces(const ForceArgs& a, cudaStream_t st) {
    int nb = blocks_for(a);
    return a.periodic ? dispatch_periodic(a, nb, st, nullptr) : dispatch_open(a, nb, st, nullptr);
}
#else
cudaError_t dispatch_periodic(const ForceArgs& a, int nblocks, cudaStream_t st, int* occ) {
    if (a.order >= 4) return launch_scap<4, true>(a, a.scap, nblocks, st, occ);
    if (a.order >= 2) return launch_scap<2, true>(a, a.scap, nblocks, st, occ);
    return launch_scap<0, true>(a, a.scap, nblocks, st, occ);
}
#endif

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

#include "hot_interact.cuh"
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
    uint32_t s = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() {
    asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
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
    template <int ORDER, bool DIP = false>
    __device__ __forceinline__ void pc(const float4 q0, const float4 q1, const float4 q2, const float* m, float eps2, const float4 qd = make_float4(0.f, 0.f, 0.f, 0.f)) {
#pragma unroll
        for (int p = 0; p < NP; ++p) pc_one<ORDER, f2, DIP>(q0, q1, q2, m, x2[p], eps2, a2[p], qd);
        if (TAIL) pc_one<ORDER, float, DIP>(q0, q1, q2, m, x1, eps2, a1, qd);
    }
};

// ---- per-warp shared-memory layout (byte offsets from the warp's base) -------------------------
template <int ORDER, bool BGV = false> struct WL {
    static constexpr int NQ = PCQ<ORDER>::v + (BGV ? 1 : 0); // background-subtracted cells: one more slot, the dipole
    static constexpr int pcst = 0;                               // 2 x [NQ][32] float4  staged cells
    static constexpr int ppst = pcst + 2 * NQ * 32 * 16;         // 2 x [32] float4      staged bodies
    static constexpr int accum = ppst + 2 * 32 * 16;             // [SMAX*4][32] double  running sums (acc, pot) per lane
    static constexpr int bytes = accum + SMAX * 4 * 32 * 8;
};

// ---- S8/S9/S10: one chunk (<= 32*SMAX sinks) of one group -----------------------------------------
// L = 1 << lgL lanes per source stream, S = ceil(nchunk / L) sinks per lane.
template <int ORDER, bool PER, int S, bool SPL, bool BGV>
__device__ __noinline__ void eval_chunk(const ForceArgs& P, const int w, const GroupRec g, const int64_t gi, const uint32_t chunk0,
                                        const uint32_t nchunk, const int lgL, const int lane) {
    using Lay = WL<ORDER, BGV>;
    constexpr int NQ = Lay::NQ, QD = PCQ<ORDER>::v; // QD: slot of the dipole (BGV)
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
        float4 dipv = make_float4(0.f, 0.f, 0.f, 0.f); // BGV: (mass - cube, dipole) of the cell being gathered
        uint32_t cnext = 0; int inext = 62, pim = 62;
        auto fetch_idx = [&](int b) { // list entries of batch b
            if (b * BATCH + lane < n) { cnext = pl[b * BATCH + lane]; if (PER) inext = pi[b * BATCH + lane]; }
        };
        auto issue = [&](int b) { // gather batch b: centre to registers, moments straight to shared memory
            if (b * BATCH + lane < n) {
                const uint32_t c = PER ? (cnext & ~HOT_COARSE_FLAG) : cnext;
                pim = inext;
                if (BGV) { // a background-subtracted cell: expansion centre = the cell's centre, mass and dipole from bgA
                    const WalkCell wc = P.wcell[c];
                    const double hh = P.size * (1.0 / 2097152.0), half = 0.5 * ldexp(P.size, -(int)(wc.w >> 27));
                    cA.zx = P.lo[0] + (double)(wc.x & 0x1fffffu) * hh + half;
                    cA.zy = P.lo[1] + (double)((wc.x >> 21) | ((wc.y & 0x3ffu) << 11)) * hh + half;
                    cA.zz = P.lo[2] + (double)((wc.y >> 10) & 0x1fffffu) * hh + half;
                    dipv = P.bgA[c];
                    cA.m0 = dipv.x;
                } else {
                    cA = P.cellA[c];
                    if (PER && (cnext & HOT_COARSE_FLAG)) cA.m0 = 0.f; // its monopole is summed in fp64 elsewhere (hot_periodic.cu)
                }
                float4* const dst = pcst + (b & 1) * NQ * BATCH + lane;
                if (ORDER >= 2) {
                    const float4* src = reinterpret_cast<const float4*>((BGV ? P.bgE2 : P.cellE2) + c);
                    cp_async16(dst + 1 * BATCH, src);
                    cp_async16(dst + 2 * BATCH, src + 1);
                }
                if (ORDER >= 4) {
                    const float4* src = reinterpret_cast<const float4*>((BGV ? P.bgM34 : P.cellM34) + c);
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
                if (BGV) st[QD * 32 + lane] = make_float4(dipv.y, dipv.z, dipv.w, 0.f);
            }
            if (ORDER >= 2) cp_async_wait_all();
            __syncwarp();
            if (b + 1 < nb) { issue(b + 1); fetch_idx(b + 2); } // in flight during the arithmetic below
            if (ORDER < 4) { // the next source's record is read while the current one is evaluated
                int j = strm;
                float4 n0 = st[j < cnt ? j : 0], n1 = n0, n2 = n0, nd = n0;
                if (ORDER >= 2) { n1 = st[32 + (j < cnt ? j : 0)]; n2 = st[64 + (j < cnt ? j : 0)]; }
                if (BGV) nd = st[QD * 32 + (j < cnt ? j : 0)];
                if (S >= UNROLL2_S) { // two sources per trip: the sums stay in their registers (no copies at the loop end)
#pragma unroll 2
                while (j < cnt) {
                    const float4 q0 = n0, q1 = n1, q2 = n2, qd = nd;
                    j += K;
                    const int jn = j < cnt ? j : strm;
                    n0 = st[jn];
                    if (ORDER >= 2) { n1 = st[32 + jn]; n2 = st[64 + jn]; }
                    if (BGV) nd = st[QD * 32 + jn];
                    sk.template pc<ORDER, BGV>(q0, q1, q2, nullptr, eps2, qd);
                }
                } else {
#pragma unroll 1
                while (j < cnt) {
                    const float4 q0 = n0, q1 = n1, q2 = n2, qd = nd;
                    j += K;
                    const int jn = j < cnt ? j : strm;
                    n0 = st[jn];
                    if (ORDER >= 2) { n1 = st[32 + jn]; n2 = st[64 + jn]; }
                    if (BGV) nd = st[QD * 32 + jn];
                    sk.template pc<ORDER, BGV>(q0, q1, q2, nullptr, eps2, qd);
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
                    sk.template pc<ORDER, BGV>(q0, q1, q2, m, eps2, BGV ? st[QD * 32 + j] : make_float4(0.f, 0.f, 0.f, 0.f));
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
            if (BGV) { // the background-subtracted cells' share goes to farc (fp64, key order): the launch over the plain
                       // near field adds it to its own fp64 sums and rounds once
                if (sk.me[i] >= 0) {
                    double4* const f = reinterpret_cast<double4*>(P.out_farc) + (g.first + sk.me[i]);
                    double4 r = *f;
                    r.x += A[i][0]; r.y += A[i][1]; r.z += A[i][2]; r.w += A[i][3];
                    *f = r;
                }
            } else if (sk.me[i] >= 0) {
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
template <int ORDER, bool PER, bool SPL, bool BGV>
__device__ __forceinline__ void run_chunk(const ForceArgs& P, const int w, const GroupRec g, const int64_t gi, const uint32_t c0,
                                          const uint32_t nc, const int lgL, const int lane) {
    const int S = (int)((nc + (1u << lgL) - 1) >> lgL);
    if (S <= 1) eval_chunk<ORDER, PER, 1, SPL, BGV>(P, w, g, gi, c0, nc, lgL, lane);
    else if (S == 2) eval_chunk<ORDER, PER, 2, SPL, BGV>(P, w, g, gi, c0, nc, lgL, lane);
    else if (S == 3) eval_chunk<ORDER, PER, 3, SPL, BGV>(P, w, g, gi, c0, nc, lgL, lane);
    else if (S == 4) eval_chunk<ORDER, PER, 4, SPL, BGV>(P, w, g, gi, c0, nc, lgL, lane);
    else if (S == 5) eval_chunk<ORDER, PER, 5, SPL, BGV>(P, w, g, gi, c0, nc, lgL, lane);
    else eval_chunk<ORDER, PER, 6, SPL, BGV>(P, w, g, gi, c0, nc, lgL, lane);
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

template <int ORDER, bool PER, bool SPL, bool BGV>
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
        run_chunk<ORDER, PER, SPL, BGV>(P, w, P.group[gi], gi, it.y, it.z, (int)it.w, lane);
    }
}

template <int ORDER, bool PER, bool SPL, bool BGV = false> static cudaError_t launch_one(const ForceArgs& a, cudaStream_t st) {
    constexpr int smem = WL<ORDER, BGV>::bytes * WARPS_PER_BLOCK;
    static int nblocks = 0;
    if (!nblocks) {
        cudaError_t e = cudaFuncSetAttribute(forces_kernel<ORDER, PER, SPL, BGV>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        int dev = 0, nsm = 0, occ = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, forces_kernel<ORDER, PER, SPL, BGV>, WARPS_PER_BLOCK * 32, smem);
        if (e != cudaSuccess) return e;
        nblocks = nsm * (occ < 1 ? 1 : occ);
    }
    HOT_LAUNCHED(1);
    forces_kernel<ORDER, PER, SPL, BGV><<<nblocks, WARPS_PER_BLOCK * 32, smem, st>>>(a);
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
    if (a.bgv) { // the flagged cells of a background-subtracted walk (hot_bg.cu): about their centres, with the dipole
        if (a.order >= 4) return launch_one<4, true, false, true>(a, st);
        if (a.order >= 2) return launch_one<2, true, false, true>(a, st);
        return launch_one<0, true, false, true>(a, st);
    }
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

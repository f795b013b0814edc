// hot_forces.cu -- S7 walk fused with S8 particle-particle and S9 particle-cell kernels, S10 scatter.
//
// One warp owns one sink group at a time (persistent grid, dynamic group counter).
//
// Walk (S7).  The warp traverses the tree cooperatively: it pops up to 32 cells from a
// shared-memory stack, every lane applies the multipole acceptance criterion to one cell (integer
// geometry, one IEEE double multiply and compare -- DESIGN.md R-7), and ballots sort the cells into
//   accepted      -> cell index appended to the particle-cell list  (shared memory),
//   rejected leaf -> its body indices appended to the particle-particle list (shared memory),
//   else          -> its children pushed on the stack.
// The walk is one function shared by every sink-blocking variant (walk_some): its state lives in
// shared memory, it returns when a list holds LIST_DRAIN entries or the traversal is finished, the
// caller evaluates the full batches and calls it again.  The lists never leave shared memory.
//
// Evaluation (S8, S9) -- the m x n blocking of PAPER.md:162-164.  The 32 lanes are split into
// K = 32/L "source streams" of L lanes.  Every stream holds ALL sinks of the group in registers
// (S = ceil(n/L) <= SMAX per lane) and takes every K-th source of a 32-source batch, read from shared
// memory as broadcast 128-bit loads.  L is the smallest power of two with ceil(n/L) <= SMAX, so at
// most L-1 of the L*S sink slots idle whatever the group size; the K partial sums are combined
// with shuffles once per group.  Batches are staged one ahead of the arithmetic: cell centres and
// bodies are prefetched into registers (they need the fp64 shift to group-relative coordinates),
// moments go global -> shared directly with cp.async.
//
// Arithmetic: interactions in fp32 (FFMA + MUFU.RSQ), coordinates relative to the group centre
// (formed in fp64 when a source is staged), per-lane partial sums of <= 32 sources in fp32, running
// sums in fp64.
#include "hot_internal.h"

#define FULL 0xffffffffu
#define BATCH 32               // sources per staged batch
#define LIST_DRAIN 256         // evaluate when the cell / body list holds this many entries
#define LIST_CAP (LIST_DRAIN + 32)
#define RUN_DRAIN 32           // ... or the list of rejected leaves (body runs) this many
#define RUN_CAP (RUN_DRAIN + 32)
#define WARPS_PER_BLOCK 4
#define SMAX 4                 // sinks per lane

template <bool PER> struct StackCap { static constexpr int v = 512; }; // ring entries (runs of <= 8 sibling cells), a power of two
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
// Staged cell j of a batch: float4 slot q of the record sits at st[q*32 + j] (slot-major, so the
// K streams of a warp read K consecutive float4 -- no bank conflicts for any K):
//   slot 0: (zx, zy, zz, M0)  centre of mass relative to the group origin
//   slot 1: (xx, xy, xz, yy)  slot 2: (yz, zz, t2, -)                        ORDER >= 2
//   slots 3..11: M3 (10) M4 (15) t3 (3) T4 (6: xx xy xz yy yz zz) t4 (1) pad   ORDER >= 4
template <int ORDER, int S>
__device__ __forceinline__ void pc_eval(const float4* __restrict__ st, const int j, const float (&x)[S][3], float eps2,
                                        float (&a)[S][4]) {
    const float4 q0 = st[j];
    float4 q1, q2;
    if (ORDER >= 2) { q1 = st[32 + j]; q2 = st[64 + j]; }
    float m[ORDER >= 4 ? 36 : 1];
    if (ORDER >= 4) {
#pragma unroll
        for (int k = 0; k < 9; ++k) {
            const float4 t = st[(3 + k) * 32 + j];
            m[4 * k] = t.x; m[4 * k + 1] = t.y; m[4 * k + 2] = t.z; m[4 * k + 3] = t.w;
        }
    }
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
        // quadrupole.  p5 = 1.5 u^-5/2, p7 = -7.5 u^-7/2:
        //   phi = -M0 ri + 0.5 t2 ri3 - p5 Q2;  a = R (-M0 ri3 + t2 p5 + p7 Q2) + 2 p5 (M2 R)
        const float p5 = ri3 * (1.5f * ri2), p7 = p5 * (-5.0f * ri2);
        const float Mx = fmaf(q1.x, Rx, fmaf(q1.y, Ry, q1.z * Rz));
        const float My = fmaf(q1.y, Rx, fmaf(q1.w, Ry, q2.x * Rz));
        const float Mz = fmaf(q1.z, Rx, fmaf(q2.x, Ry, q2.y * Rz));
        const float Q2 = fmaf(Mx, Rx, fmaf(My, Ry, Mz * Rz));
        const float t2 = q2.z;
        float cR = fmaf(p7, Q2, fmaf(t2, p5, -q0.w * ri3));
        float ph = fmaf(0.5f * t2, ri3, fmaf(-p5, Q2, -q0.w * ri));
        const float D2 = p5 + p5;
        float vx = D2 * Mx, vy = D2 * My, vz = D2 * Mz;
        if (ORDER >= 4) {
            const float ri5 = ri3 * ri2, ri7 = ri5 * ri2, ri9 = ri7 * ri2, ri11 = ri9 * ri2;
            const float D2f = 3.0f * ri5, D3 = -15.0f * ri7, D4 = 105.0f * ri9, D5 = -945.0f * ri11;
            const float* m3 = m;          // 10
            const float* m4 = m + 10;     // 15
            const float* t3 = m + 25;     // 3
            const float* T4 = m + 28;     // 6: xx xy xz yy yz zz
            const float t4 = m[34];
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
            ph = fmaf(D3 * (1.0f / 6.0f), S3, fmaf(0.5f * D2f, T3, ph));
            ph = fmaf(-D4 * (1.0f / 24.0f), S4, fmaf(-0.25f * D3, Q4, fmaf(-0.125f * D2f, t4, ph)));
            // a3 = -[D4 S3 R + 3 D3 V3 + 3 D3 T3 R + 3 D2 t3]/6
            // a4 = [D5 S4 R + 4 D4 W4 + 6 D4 Q4 R + 12 D3 U + 3 D3 t4 R]/24
            cR = fmaf(-D4 * (1.0f / 6.0f), S3, fmaf(-0.5f * D3, T3, cR));
            cR = fmaf(D5 * (1.0f / 24.0f), S4, fmaf(0.25f * D4, Q4, fmaf(0.125f * D3, t4, cR)));
            const float hD3n = -0.5f * D3, hD2n = -0.5f * D2f, sD4 = D4 * (1.0f / 6.0f), hD3p = 0.5f * D3;
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

// ---- per-warp shared-memory layout (byte offsets from the warp's base) -------------------------
struct WalkState {         // traversal state between two walk_some calls
    int head, top, gtop;   // ring buffer of pending cells: first entry, count; entries spilled to the global arena
    int npc, nrun;         // pending accepted cells / pending body runs (rejected leaves)
    int next_img;          // periodic: next image to seed; open: 0 before the root is seeded
    uint32_t nspill;
    unsigned long long nvisit, Lpc, Lpp;
};
template <int ORDER, bool PER> struct WL {
    static constexpr int NQ = PCQ<ORDER>::v;
    static constexpr int SC = StackCap<PER>::v;
    static constexpr int pcst = 0;                               // 2 x [NQ][32] float4  staged cells
    static constexpr int ppst = pcst + 2 * NQ * 32 * 16;         // 2 x [32] float4      staged bodies
    static constexpr int stack = ppst + 2 * 32 * 16;             // [SC] u32             pending cells (ring, SC a power of two)
    static constexpr int pcidx = stack + SC * 4;                 // [LIST_CAP] u32       accepted cells
    static constexpr int ppidx = pcidx + LIST_CAP * 4;           // [LIST_CAP] u32       bodies to evaluate
    static constexpr int runf = ppidx + LIST_CAP * 4;            // [RUN_CAP] u32        first body of a rejected leaf
    static constexpr int runn = runf + RUN_CAP * 4;              // [RUN_CAP] u32        its body count
    static constexpr int state = runn + RUN_CAP * 4;             // WalkState (64 B reserved)
    static constexpr int accum = state + 64;                     // [SMAX*4][32] double  running sums (acc, pot) per lane
    static constexpr int stimg = accum + SMAX * 4 * 32 * 8;      // periodic: image id per entry (u8)
    static constexpr int pcimg = stimg + (PER ? SC : 0);
    static constexpr int ppimg = pcimg + (PER ? LIST_CAP : 0);
    static constexpr int runimg = ppimg + (PER ? LIST_CAP : 0);
    static constexpr int bytes = (runimg + (PER ? RUN_CAP : 0) + 15) & ~15;
};
static_assert(sizeof(WalkState) <= 64, "WalkState must fit its shared-memory slot");

// ---- S7: advance the traversal of group cell `gcell` until a list is full or the tree is done ----
// Returns true when the traversal is finished (warp-uniform).
template <int ORDER, bool PER>
__device__ __noinline__ bool walk_some(const ForceArgs& P, const int w, const int lane, const uint32_t gcell, uint32_t* gstack) {
    using Lay = WL<ORDER, PER>;
    constexpr int SC = Lay::SC;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    unsigned char* const base = smem_raw + (size_t)w * Lay::bytes;
    uint32_t* const stack = reinterpret_cast<uint32_t*>(base + Lay::stack);
    uint32_t* const pcidx = reinterpret_cast<uint32_t*>(base + Lay::pcidx);
    uint32_t* const runf = reinterpret_cast<uint32_t*>(base + Lay::runf);
    uint32_t* const runn = reinterpret_cast<uint32_t*>(base + Lay::runn);
    WalkState* const wsm = reinterpret_cast<WalkState*>(base + Lay::state);
    uint8_t* const stimg = base + Lay::stimg;
    uint8_t* const pcimg = base + Lay::pcimg;
    uint8_t* const runimg = base + Lay::runimg;

    const uint32_t lt = (1u << lane) - 1u;
    // group cube on the integer grid
    const WalkCell gw = P.wcell[gcell];
    const int gs = 1 << (HOT_MAXLEVEL - (int)(gw.w >> 27));
    const int gox = (int)(gw.x & 0x1fffffu), goy = (int)((gw.x >> 21) | ((gw.y & 0x3ffu) << 11)), goz = (int)((gw.y >> 10) & 0x1fffffu);
    const double theta2 = P.theta2;
    // Pending work sits in a ring buffer used as a deque.  An entry is a run of sibling cells
    // (first cell | (count-1) << 28, count <= 8): opening a cell pushes ONE entry.  While the ring is
    // short the warp pops the OLDEST entries (breadth-first, which keeps the frontier wide and the
    // 32 lanes busy); once it holds DEQ_DFS entries it pops the NEWEST (depth-first, bounded growth).
    constexpr int M = SC - 1, DEQ_DFS = SC / 4;
    int head = wsm->head, top = wsm->top, gtop = wsm->gtop, npc = wsm->npc, nrun = wsm->nrun, next_img = wsm->next_img;
    uint32_t nspill = 0, nvisit = 0, dLpc = 0;
    unsigned long long dLpp = 0;
    bool done = false;
    constexpr int NIMG = PER ? 125 : 1;
    while (npc < LIST_DRAIN && nrun < RUN_DRAIN) {
        if (top == 0) {
            if (gtop > 0) { // refill from the global arena
                const int mv = gtop > SC / 2 ? SC / 2 : gtop;
                for (int t = lane; t < mv; t += 32) {
                    stack[(head + t) & M] = gstack[gtop - mv + t];
                    if (PER) stimg[(head + t) & M] = (uint8_t)gstack[P.gstack_cap + gtop - mv + t];
                }
                gtop -= mv; top = mv;
            } else if (next_img < NIMG) { // seed: the root once per image (lane = image)
                const int im = next_img + lane;
                if (im < NIMG) { stack[(head + lane) & M] = 0u; if (PER) stimg[(head + lane) & M] = (uint8_t)im; }
                top = min(32, NIMG - next_img);
                next_img += top;
            } else { done = true; break; }
            __syncwarp();
        }
        if (SC - top < 32) { // no room for 32 pushes: spill the oldest entries to the global arena, keep 128
            const int keep = 128, mv = top - keep;
            if ((int64_t)gtop + mv > P.gstack_cap) { if (lane == 0) atomicOr(P.errflag, 4); top = 0; gtop = 0; next_img = NIMG; done = true; break; }
            for (int t = lane; t < mv; t += 32) {
                gstack[gtop + t] = stack[(head + t) & M];
                if (PER) gstack[P.gstack_cap + gtop + t] = stimg[(head + t) & M]; // image ids: second half of the arena
            }
            __syncwarp();
            gtop += mv; head = (head + mv) & M; top = keep; ++nspill;
        }
        // take whole entries while they hold <= 32 cells in total, one cell per lane
        uint32_t c = 0; int im = PER ? 62 : 0, nt;
        {
            const bool dfs = top >= DEQ_DFS;
            const int at = dfs ? (head + top - 1 - lane) & M : (head + lane) & M;
            uint32_t e = 0; int eim = 62, ecnt = 0;
            if (lane < top) { e = stack[at]; if (PER) eim = stimg[at]; ecnt = (int)(e >> 28) + 1; }
            int incl = ecnt;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(FULL, incl, o); if (lane >= o) incl += y; }
            const bool take = lane < top && incl <= 32;
            const int ne = __popc(__ballot_sync(FULL, take));                 // >= 1: an entry holds <= 8 cells
            nt = __shfl_sync(FULL, incl, ne - 1);
            const int excl = incl - ecnt;
            const uint32_t starts = __reduce_or_sync(FULL, take ? (1u << excl) : 0u);
            const int src = __popc(starts & ((2u << lane) - 1u)) - 1;         // entry that holds this lane's cell
            const int srcl = src < 0 ? 0 : src;
            const uint32_t eb = __shfl_sync(FULL, e & 0x0fffffffu, srcl);
            const int ex = __shfl_sync(FULL, excl, srcl);
            if (PER) im = __shfl_sync(FULL, eim, srcl);
            c = eb + (uint32_t)(lane - ex);
            if (!dfs) head = (head + ne) & M;
            top -= ne;
        }
        const bool v = lane < nt;
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
        const bool acc = v && (s2 < theta2 * __ull2double_rn(d2));
        const bool self = v && c == gcell && (!PER || im == 62);
        const bool rej_leaf = v && !acc && leaf && !self;
        const bool open = v && !acc && !leaf && !self;
        // accepted cells -> P-C list; rejected leaves -> run list; opened cells -> their child run into the ring
        const uint32_t macc = __ballot_sync(FULL, acc), mrej = __ballot_sync(FULL, rej_leaf), mopen = __ballot_sync(FULL, open);
        if (acc) { const int p = npc + __popc(macc & lt); pcidx[p] = c; if (PER) pcimg[p] = (uint8_t)im; }
        npc += __popc(macc); dLpc += __popc(macc);
        if (rej_leaf) { const int p = nrun + __popc(mrej & lt); runf[p] = wc.z; runn[p] = cnt; if (PER) runimg[p] = (uint8_t)im; }
        nrun += __popc(mrej);
        if (mrej) {
            uint32_t nb = rej_leaf ? cnt : 0u;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) nb += __shfl_xor_sync(FULL, nb, o);
            dLpp += nb;
        }
        if (open) {
            const int p = (head + top + __popc(mopen & lt)) & M;
            stack[p] = wc.z | ((cnt - 1u) << 28);
            if (PER) stimg[p] = (uint8_t)im;
        }
        top += __popc(mopen);
        __syncwarp();
    }
    if (!done && top == 0 && gtop == 0 && next_img >= NIMG) done = true;
    if (lane == 0) {
        wsm->head = head; wsm->top = top; wsm->gtop = gtop; wsm->npc = npc; wsm->nrun = nrun; wsm->next_img = next_img;
        wsm->nspill += nspill; wsm->nvisit += nvisit; wsm->Lpc += dLpc; wsm->Lpp += dLpp;
    }
    __syncwarp();
    return done;
}

// ---- S8/S9/S10: one chunk (<= 32*SMAX sinks) of one group -----------------------------------------
// L = 1 << lgL lanes per source stream, S = ceil(nchunk / L) sinks per lane.
template <int ORDER, bool PER, int S>
__device__ __noinline__ void process_chunk(const ForceArgs& P, const int w, const GroupRec g, const uint32_t chunk0,
                                           const uint32_t nchunk, const int lgL, uint32_t* gstack, const int lane) {
    using Lay = WL<ORDER, PER>;
    constexpr int NQ = Lay::NQ;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    unsigned char* const base = smem_raw + (size_t)w * Lay::bytes;
    float4* const pcst = reinterpret_cast<float4*>(base + Lay::pcst);
    float4* const ppst = reinterpret_cast<float4*>(base + Lay::ppst);
    uint32_t* const pcidx = reinterpret_cast<uint32_t*>(base + Lay::pcidx);
    uint32_t* const ppidx = reinterpret_cast<uint32_t*>(base + Lay::ppidx);
    const uint32_t* const runf = reinterpret_cast<const uint32_t*>(base + Lay::runf);
    const uint32_t* const runn = reinterpret_cast<const uint32_t*>(base + Lay::runn);
    WalkState* const wsm = reinterpret_cast<WalkState*>(base + Lay::state);
    double* const As = reinterpret_cast<double*>(base + Lay::accum) + lane; // this lane's running sums: As[(4 i + k) * 32]
    uint8_t* const pcimg = base + Lay::pcimg;
    uint8_t* const ppimg = base + Lay::ppimg;
    const uint8_t* const runimg = base + Lay::runimg;

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
    float x[S][3];
    int me[S];
    float a[S][4];
#pragma unroll
    for (int i = 0; i < S; ++i) {
        const uint32_t loc = (uint32_t)(i * L + sl);
        me[i] = loc < nchunk ? (int)(chunk0 + loc) : -1;
        const float4 b = P.body[g.first + (loc < nchunk ? chunk0 + loc : 0u)];
        x[i][0] = (float)((double)b.x - ox); x[i][1] = (float)((double)b.y - oy); x[i][2] = (float)((double)b.z - oz);
#pragma unroll
        for (int k = 0; k < 4; ++k) { a[i][k] = 0.0f; As[(4 * i + k) * 32] = 0.0; }
    }
    const float eps2 = P.eps2;
    // fp32 partials a[] are added to the fp64 running sums (shared memory, lane-private) after at
    // most ~32 sources per lane and at the end of every drain, so a[] is dead across the walk
    int nacc = 0;
    auto flush = [&]() {
#pragma unroll
        for (int i = 0; i < S; ++i)
#pragma unroll
            for (int k = 0; k < 4; ++k) { As[(4 * i + k) * 32] += (double)a[i][k]; a[i][k] = 0.0f; }
        nacc = 0;
    };
    auto shift_of = [&](int im, double& shx, double& shy, double& shz) {
        shx = (double)(im / 25 - 2) * P.size; shy = (double)((im / 5) % 5 - 2) * P.size; shz = (double)(im % 5 - 2) * P.size;
    };

    // ---- S8 driver: evaluate bodies ppidx[0..n) (n a multiple of 32 except in the final drain) ----
    auto drain_pp = [&](const int n) {
        const int nb = (n + BATCH - 1) / BATCH;
        float4 pb = make_float4(0.f, 0.f, 0.f, 0.f);
        int pim = 62;
        auto fetch = [&](int b) {
            if (b * BATCH + lane < n) {
                pb = P.body[ppidx[b * BATCH + lane]];
                if (PER) pim = ppimg[b * BATCH + lane];
            }
        };
        fetch(0);
        for (int b = 0; b < nb; ++b) {
            const int cnt = min(BATCH, n - b * BATCH);
            float4* const st = ppst + (b & 1) * BATCH;
            if (lane < cnt) {
                double shx = 0, shy = 0, shz = 0;
                if (PER) shift_of(pim, shx, shy, shz);
                st[lane] = make_float4((float)((double)pb.x + shx - ox), (float)((double)pb.y + shy - oy),
                                       (float)((double)pb.z + shz - oz), pb.w);
            }
            __syncwarp();
            if (b + 1 < nb) fetch(b + 1); // in flight during the arithmetic below
#pragma unroll 1
            for (int j = strm; j < cnt; j += K) pp_eval<S>(st[j], x, eps2, a);
            nacc += (cnt + K - 1) >> lgK;
            if (nacc >= 32) flush();
        }
        if (nacc > 0) flush();
        __syncwarp();
    };
    // ---- S9 driver: evaluate cells pcidx[0..n) ------------------------------------------------------
    auto drain_pc = [&](const int n) {
        const int nb = (n + BATCH - 1) / BATCH;
        CellA cA;
        cA.zx = cA.zy = cA.zz = 0.0; cA.m0 = 0.f; cA.t2 = 0.f;
        int pim = 62;
        auto issue = [&](int b) {
            if (b * BATCH + lane < n) {
                const uint32_t c = pcidx[b * BATCH + lane];
                if (PER) pim = pcimg[b * BATCH + lane];
                cA = P.cellA[c];
                float4* const dst = pcst + (b & 1) * NQ * BATCH + lane;
                if (ORDER >= 2) {
                    const float4* src = reinterpret_cast<const float4*>(P.cellM2 + c);
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
        issue(0);
        for (int b = 0; b < nb; ++b) {
            const int cnt = min(BATCH, n - b * BATCH);
            float4* const st = pcst + (b & 1) * NQ * BATCH;
            if (lane < cnt) {
                double shx = 0, shy = 0, shz = 0;
                if (PER) shift_of(pim, shx, shy, shz);
                st[lane] = make_float4((float)(cA.zx + shx - ox), (float)(cA.zy + shy - oy), (float)(cA.zz + shz - oz), cA.m0);
            }
            if (ORDER >= 2) cp_async_wait_all();
            __syncwarp();
            if (b + 1 < nb) issue(b + 1);
#pragma unroll 1
            for (int j = strm; j < cnt; j += K) pc_eval<ORDER, S>(st, j, x, eps2, a);
            nacc += (cnt + K - 1) >> lgK;
            if (nacc >= 32) flush();
        }
        if (nacc > 0) flush();
        __syncwarp();
    };

    if (lane == 0) {
        WalkState z;
        z.head = z.top = z.gtop = z.npc = z.nrun = z.next_img = 0; z.nspill = 0; z.nvisit = 0; z.Lpc = 0; z.Lpp = g.count;
        *wsm = z;
    }
    // the group's own bodies (the "self block"): the walk skips the group cell itself
    for (uint32_t j0 = 0; j0 < g.count; j0 += BATCH) {
        const int cnt = (int)min((uint32_t)BATCH, g.count - j0);
        if (lane < cnt) {
            const float4 b = P.body[g.first + j0 + lane];
            ppst[lane] = make_float4((float)((double)b.x - ox), (float)((double)b.y - oy), (float)((double)b.z - oz), b.w);
        }
        __syncwarp();
#pragma unroll 1
        for (int j = strm; j < cnt; j += K) pp_eval_self<S>(ppst[j], (int)j0 + j, me, x, eps2, a);
        __syncwarp();
    }
    flush();

    int npp = 0; // bodies waiting in ppidx
    bool done;
    do {
        done = walk_some<ORDER, PER>(P, w, lane, g.cell, gstack);
        int npc = wsm->npc;
        const int nrun = wsm->nrun;
        __syncwarp();
        // accepted cells
        {
            const int nd = done ? npc : (npc >= LIST_DRAIN ? (npc & ~(BATCH - 1)) : 0);
            if (nd > 0) {
                drain_pc(nd);
                npc -= nd;
                uint32_t t = 0; uint8_t ti = 0;
                if (lane < npc) { t = pcidx[nd + lane]; if (PER) ti = pcimg[nd + lane]; }
                __syncwarp();
                if (lane < npc) { pcidx[lane] = t; if (PER) pcimg[lane] = ti; }
            }
        }
        // rejected leaves: expand their body runs into the body list, evaluate its full batches
        if (done || nrun >= RUN_DRAIN) {
            int r = 0; uint32_t j0 = 0;
            while (true) {
                while (r < nrun && npp < LIST_DRAIN) {
                    const uint32_t f = runf[r], n = runn[r];
                    const uint32_t k = min((uint32_t)BATCH, n - j0);
                    if ((uint32_t)lane < k) { ppidx[npp + lane] = f + j0 + lane; if (PER) ppimg[npp + lane] = runimg[r]; }
                    npp += (int)k; j0 += k;
                    if (j0 >= n) { ++r; j0 = 0; }
                }
                __syncwarp();
                const bool last = r >= nrun;
                const int nd = (last && done) ? npp : (npp >= LIST_DRAIN ? (npp & ~(BATCH - 1)) : 0);
                if (nd > 0) {
                    drain_pp(nd);
                    npp -= nd;
                    uint32_t t = 0; uint8_t ti = 0;
                    if (lane < npp) { t = ppidx[nd + lane]; if (PER) ti = ppimg[nd + lane]; }
                    __syncwarp();
                    if (lane < npp) { ppidx[lane] = t; if (PER) ppimg[lane] = ti; }
                    __syncwarp();
                }
                if (last) break;
            }
            if (lane == 0) wsm->nrun = 0;
        }
        if (lane == 0) wsm->npc = npc;
        __syncwarp();
    } while (!done);
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
    // S10: results to the caller's particle order
    if (strm == 0) {
#pragma unroll
        for (int i = 0; i < S; ++i) {
            if (me[i] >= 0) {
                const uint32_t o = P.perm[g.first + me[i]];
                P.acc[3 * (int64_t)o] = (float)A[i][0];
                P.acc[3 * (int64_t)o + 1] = (float)A[i][1];
                P.acc[3 * (int64_t)o + 2] = (float)A[i][2];
                if (P.pot) P.pot[o] = (float)A[i][3];
            }
        }
    }
}

template <int ORDER, bool PER>
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32, ORDER >= 4 ? 3 : 4) forces_kernel(const __grid_constant__ ForceArgs P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const WalkState* const wsm = reinterpret_cast<const WalkState*>(smem_raw + (size_t)w * WL<ORDER, PER>::bytes + WL<ORDER, PER>::state);
    const int64_t gwarp = (int64_t)blockIdx.x * WARPS_PER_BLOCK + w;
    uint32_t* gstack = P.gstack + gwarp * P.gstack_cap * (PER ? 2 : 1);
    unsigned long long nvisit = 0, nspill = 0, sum_pp = 0, sum_pc = 0;
    while (true) {
        unsigned int gi = 0;
        if (lane == 0) gi = atomicAdd(P.counter, 1u);
        gi = __shfl_sync(FULL, gi, 0);
        if ((int64_t)gi >= P.ngroups) break;
        const GroupRec g = P.group[gi];
        // sinks in chunks of at most 32*SMAX (only groups larger than that need more than one walk)
        for (uint32_t c0 = 0; c0 < g.count; c0 += 32 * SMAX) {
            const uint32_t nc = min((uint32_t)(32 * SMAX), g.count - c0);
            int lgL = 0;
            while (((nc + (1u << lgL) - 1) >> lgL) > SMAX) ++lgL;
            const int S = (int)((nc + (1u << lgL) - 1) >> lgL);
            if (S <= 1) process_chunk<ORDER, PER, 1>(P, w, g, c0, nc, lgL, gstack, lane);
            else if (S == 2) process_chunk<ORDER, PER, 2>(P, w, g, c0, nc, lgL, gstack, lane);
            else if (S == 3) process_chunk<ORDER, PER, 3>(P, w, g, c0, nc, lgL, gstack, lane);
            else process_chunk<ORDER, PER, 4>(P, w, g, c0, nc, lgL, gstack, lane);
            if (lane == 0) { nvisit += wsm->nvisit; nspill += wsm->nspill; }
        }
        if (lane == 0) { // every chunk walks the same lists: the last chunk's counts are the group's
            const uint64_t Lpc = wsm->Lpc, Lpp = wsm->Lpp;
            P.glpc[gi] = Lpc; P.glpp[gi] = Lpp;
            sum_pp += (unsigned long long)g.count * Lpp; sum_pc += (unsigned long long)g.count * Lpc;
        }
        __syncwarp();
    }
    if (lane == 0) {
        atomicAdd(&P.stat[0], nvisit); atomicAdd(&P.stat[1], nspill);
        atomicAdd(&P.stat[2], sum_pp); atomicAdd(&P.stat[3], sum_pc);
    }
}

template <int ORDER, bool PER> static cudaError_t launch_one(const ForceArgs& a, int nblocks, cudaStream_t st, int* occ_out) {
    constexpr int smem = WL<ORDER, PER>::bytes * WARPS_PER_BLOCK;
    cudaError_t e = cudaFuncSetAttribute(forces_kernel<ORDER, PER>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    if (occ_out) {
        int occ = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, forces_kernel<ORDER, PER>, WARPS_PER_BLOCK * 32, smem);
        *occ_out = occ;
        return e;
    }
    HOT_LAUNCHED(1);
    forces_kernel<ORDER, PER><<<nblocks, WARPS_PER_BLOCK * 32, smem, st>>>(a);
    return cudaGetLastError();
}
#ifndef HOT_FORCES_PERIODIC_TU
cudaError_t dispatch_open(const ForceArgs& a, int nblocks, cudaStream_t st, int* occ) {
    if (a.order >= 4) return launch_one<4, false>(a, nblocks, st, occ);
    if (a.order >= 2) return launch_one<2, false>(a, nblocks, st, occ);
    return launch_one<0, false>(a, nblocks, st, occ);
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
    (void)scap;
    ForceArgs a{}; a.order = order; a.periodic = periodic;
    return blocks_for(a) * WARPS_PER_BLOCK;
}
cudaError_t launch_forces(const ForceArgs& a, cudaStream_t st) {
    int nb = blocks_for(a);
    return a.periodic ? dispatch_periodic(a, nb, st, nullptr) : dispatch_open(a, nb, st, nullptr);
}
#else
cudaError_t dispatch_periodic(const ForceArgs& a, int nblocks, cudaStream_t st, int* occ) {
    if (a.order >= 4) return launch_one<4, true>(a, nblocks, st, occ);
    if (a.order >= 2) return launch_one<2, true>(a, nblocks, st, occ);
    return launch_one<0, true>(a, nblocks, st, occ);
}
#endif

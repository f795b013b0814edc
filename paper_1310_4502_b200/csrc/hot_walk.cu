// hot_walk.cu -- S7: the per-sink-group tree walk that emits the interaction lists.
//
// One warp owns one sink group at a time (persistent grid, dynamic group counter).  The warp
// traverses the tree cooperatively: it pops up to 32 cells from a shared-memory deque, every lane
// applies the multipole acceptance criterion to one cell (integer geometry and an integer threshold
// per level that reproduces the one IEEE double multiply and compare of DESIGN.md R-7 exactly), and
// ballots sort the cells into
//   accepted      -> cell index appended to the group's particle-cell list,
//   rejected leaf -> its body run (first, count) appended to the group's particle-particle list
//                    (expanded to one body index per entry when the list is moved to the arena),
//   else          -> its run of children pushed on the deque.
// ONE pass: a group's lists are first written to the warp's private staging area (global memory,
// L2-resident); when the walk of the group is done its exact lengths are known, the warp takes a
// contiguous slice of the list arena with one atomicAdd per list and copies the lists there.
// If the arena is full the group is reported (first_fail), the host evaluates what fits and calls
// the walk again for the rest.
// The walk is integer- and latency-bound, so it runs at high occupancy (40 registers, ~2.6 KB of
// shared memory per warp: 48 warps per SM) and leaves the FP32 work to hot_forces.cu.
#include <climits>

#include "hot_internal.h"

#define FULL 0xffffffffu
#define WALK_WARPS 8   // warps per block
#define RING 512       // deque entries per warp (runs of <= 8 sibling cells); a power of two
#define WALK_MINBLK 6 // resident blocks per SM the kernel is compiled for (40 registers): the walk of one group is a chain of dependent
                      // cell-record loads, so resident warps are what hides it (3 blocks: 10.4 ms, 5: 6.6, 6: 5.2, 8 with spills: 5.2 at C2)

// At 40 registers the kernel is bound by instruction issue (ncu: issue slots 81% busy, 4.2 G warp instructions at C2), and a
// third of the inner loop was address arithmetic that ptxas re-did every trip -- the warp's number from %ctaid and %tid,
// 64-bit products with the arena strides -- because nothing of it fitted in registers.  So what a warp needs only now and
// then lives in SLOTS words behind its ring in shared memory and is RE-READ where it is used (volatile: one LDS.64 and one
// IMAD.WIDE per staged store instead of eleven instructions): the warp's arena pointers, the number of the group it is
// walking, its spill count.  4.49 -> 3.78 ms at C2, 1.42 -> 1.22 ms at 128^3 periodic; 1368 -> 1000 instructions.
enum { SLOT_SPC = 0, SLOT_SPP = 2, SLOT_IPC = 4, SLOT_IPP = 6, SLOT_VSTACK = 8, SLOT_VSTAGE = 10, SLOT_GSTACK = 12, SLOT_GROUP = 14, SLOT_NSPILL = 15, SLOTS = 16 };
#define WSLOT(T, k) (*reinterpret_cast<T volatile*>(ring + RING + (k)))

// Pending work: a ring buffer used as a deque.  An entry is a run of sibling cells
// (first cell | (count-1) << 28, count <= 8): opening a cell pushes ONE entry.  While the ring is short
// the warp pops the four OLDEST entries (breadth-first: keeps the frontier wide and the 32 lanes busy);
// once it holds RING/4 entries it pops the NEWEST (depth-first: bounded growth).  If it still fills
// up, the oldest entries spill to a per-warp arena in global memory.
// TOL: the error-bound criterion with per-interaction order (R-16) instead of the
// opening angle: a lane also reads the cell's centre of mass, radius and moment bounds and takes the cheapest of
// monopole / quadrupole / hexadecapole whose bound at the distance to the group's cube is below the tolerance; the
// order rides in bits 29-30 of the staged entry and the list is laid out monopoles | quadrupoles | hexadecapoles.
#define HOT_ORDER_SHIFT 29
// BG (periodic boxes, with the opening angle): per-cell background subtraction (R-18; Fig 2).
// K_G = the 5 x 5 x 5 block of cells of the group's level around the group.  A cell across K_G's boundary is opened;
// an accepted cell outside K_G is flagged (bit 29: it is evaluated about its centre minus the uniform cube; the list is
// laid out plain | flagged); empty octants of opened cells and the cubes of rejected leaves outside K_G go to a stack of
// VIRTUAL cubes (only the negative background), which are accepted by the same criterion or subdivided.
template <bool PER, bool TOL, bool BG>
__global__ void __launch_bounds__(WALK_WARPS * 32, WALK_MINBLK) walk_kernel(const __grid_constant__ WalkArgs P) {
    __shared__ uint32_t s_ring[WALK_WARPS][RING + SLOTS];
    __shared__ uint8_t s_img[PER ? WALK_WARPS : 1][PER ? RING : 1];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t* const ring = s_ring[w];
    uint8_t* const rimg = s_img[PER ? w : 0];
    const int64_t gwarp = (int64_t)blockIdx.x * WALK_WARPS + w;
    const uint32_t scap = (uint32_t)P.stage_cap;
    if (lane == 0) {
        WSLOT(uint32_t*, SLOT_SPC) = P.stage + gwarp * 2 * P.stage_cap;
        WSLOT(uint32_t*, SLOT_SPP) = P.stage + gwarp * 2 * P.stage_cap + P.stage_cap;
        WSLOT(uint32_t*, SLOT_GSTACK) = P.gstack + gwarp * P.gstack_cap * (PER ? 2 : 1);
        if (PER) {
            WSLOT(uint8_t*, SLOT_IPC) = P.stage_img + gwarp * 2 * P.stage_cap;
            WSLOT(uint8_t*, SLOT_IPP) = P.stage_img + gwarp * 2 * P.stage_cap + P.stage_cap;
        }
        if (BG) {
            WSLOT(uint4*, SLOT_VSTACK) = P.vstack + gwarp * P.vstack_cap;
            WSLOT(uint4*, SLOT_VSTAGE) = P.vstage + gwarp * P.vstage_cap;
        }
        WSLOT(uint32_t, SLOT_NSPILL) = 0; // touched by lane 0 only
    }
    __syncwarp();
#define spc WSLOT(uint32_t*, SLOT_SPC)       // staged cell list
#define spp WSLOT(uint32_t*, SLOT_SPP)       // staged run list
#define ipc WSLOT(uint8_t*, SLOT_IPC)        // their image numbers (periodic)
#define ipp WSLOT(uint8_t*, SLOT_IPP)
#define gstack WSLOT(uint32_t*, SLOT_GSTACK) // where the ring spills
#define vstack WSLOT(uint4*, SLOT_VSTACK)    // BG: virtual cubes to look at: (x | y<<21, y>>11 | z<<10, level, image)
#define vstage WSLOT(uint4*, SLOT_VSTAGE)    // BG: accepted virtual cubes of the group
    const uint32_t lt = (1u << lane) - 1u;
    constexpr int M = RING - 1, DEQ_DFS = RING / 4, NIMG = PER ? 125 : 1;

    while (true) {
        unsigned int q = 0;
        if (lane == 0) q = atomicAdd(P.counter, 1u);
        q = __shfl_sync(FULL, q, 0);
        if (lane == 0) WSLOT(uint32_t, SLOT_GROUP) = q; // needed again only when the walk of the group is done
        __syncwarp();
#define gi (P.g0 + (int64_t)WSLOT(uint32_t, SLOT_GROUP))
        if (gi >= P.g1 || gi > (int64_t)*(volatile int*)P.first_fail) break;
        const GroupRec g = P.group[gi];
        const uint32_t gcell = g.cell;
        // group cube on the integer grid, as corner + size and pre-added for the gap formula
        const WalkCell gw = P.wcell[gcell];
        const int gs = 1 << (HOT_MAXLEVEL - (int)(gw.w >> 27));
        const int gox = (int)(gw.x & 0x1fffffu), goy = (int)((gw.x >> 21) | ((gw.y & 0x3ffu) << 11)), goz = (int)((gw.y >> 10) & 0x1fffffu);
        const int ghx = gox + gs, ghy = goy + gs, ghz = goz + gs;
        double gcx = 0, gcy = 0, gcz = 0, gh = 0; // TOL: the group's cube as centre and half side, in the caller's units
        if (TOL) {
            const double h = P.size * (1.0 / 2097152.0);
            gcx = P.lo[0] + ((double)gox + 0.5 * gs) * h; gcy = P.lo[1] + ((double)goy + 0.5 * gs) * h; gcz = P.lo[2] + ((double)goz + 0.5 * gs) * h;
            gh = 0.5 * (double)gs * h;
        }
        uint32_t n0 = 0, n2 = 0; // TOL: accepted monopoles, quadrupoles; BG: plain, background-subtracted cells
        const int klx = gox - 2 * gs, kly = goy - 2 * gs, klz = goz - 2 * gs, khx = gox + 3 * gs, khy = goy + 3 * gs, khz = goz + 3 * gs; // BG: K_G
        uint32_t vtop = 0, npv = 0; // BG: virtual cubes on the stack / accepted
        uint32_t npc = 0, nrun = 0, nbody = 0, nvis = 0; // list lengths, bodies in the runs, cells visited
        int head = 0, top = 0, gtop = 0, next_img = 0;
        while (true) {
            bool seed = false;
            if (top == 0) {
                if (gtop > 0) { // refill from the global arena
                    const int mv = gtop > RING / 2 ? RING / 2 : gtop;
                    for (int t = lane; t < mv; t += 32) {
                        ring[(head + t) & M] = gstack[gtop - mv + t];
                        if (PER) rimg[(head + t) & M] = (uint8_t)gstack[P.gstack_cap + gtop - mv + t];
                    }
                    gtop -= mv; top = mv;
                    __syncwarp();
                } else if (next_img < NIMG) seed = true; // the root once per image (lane = image), not through the ring
                else break;
            }
            if (RING - top < 32) { // no room for 32 pushes: spill the oldest entries, keep 128 on chip
                const int keep = 128, mv = top - keep;
                if ((int64_t)gtop + mv > P.gstack_cap) { if (lane == 0) atomicOr(P.errflag, 4); break; }
                for (int t = lane; t < mv; t += 32) {
                    gstack[gtop + t] = ring[(head + t) & M];
                    if (PER) gstack[P.gstack_cap + gtop + t] = rimg[(head + t) & M]; // image ids: second half of the arena
                }
                __syncwarp();
                gtop += mv; head = (head + mv) & M; top = keep;
                if (lane == 0) WSLOT(uint32_t, SLOT_NSPILL) = WSLOT(uint32_t, SLOT_NSPILL) + 1u;
            }
            // Up to four entries per step, eight lanes each: lane (sub, ch) = (lane / 8, lane % 8) takes child ch of entry sub.
            // An internal cell of these trees has 7.5 children on average, so the fixed mapping idles few lanes and needs no
            // scan over the entries' child counts (a third of the loop's instructions with the exact packing).
            uint32_t c = 0; int im = PER ? 62 : 0; bool v;
            if (seed) {
                im = PER ? next_img + lane : 0;
                v = next_img + lane < NIMG;
                next_img += 32;
            } else {
                const bool dfs = top >= DEQ_DFS;
                const int ne = min(top, 4), sub = lane >> 3, ch = lane & 7;
                const int at = dfs ? (head + top - 1 - sub) & M : (head + sub) & M;
                uint32_t e = 0;
                v = sub < ne;
                if (v) { e = ring[at]; if (PER) im = rimg[at]; }
                v = v && ch <= (int)(e >> 28);
                c = (e & 0x0fffffffu) + (uint32_t)ch;
                if (!dfs) head = (head + ne) & M;
                top -= ne;
            }
            const int nt = __popc(__ballot_sync(FULL, v));
            __syncwarp();
            WalkCell wc = {0, 0, 0, 0};
            if (v) wc = P.wcell[c];
            nvis += nt;
            const int lev = (int)(wc.w >> 27);
            const uint32_t cnt = wc.w & 0x7ffffffu;
            const bool leaf = (wc.y >> 31) != 0;
            int cx = (int)(wc.x & 0x1fffffu), cy = (int)((wc.x >> 21) | ((wc.y & 0x3ffu) << 11)), cz = (int)((wc.y >> 10) & 0x1fffffu);
            if (PER) { cx += (im / 25 - 2) << HOT_MAXLEVEL; cy += ((im / 5) % 5 - 2) << HOT_MAXLEVEL; cz += (im % 5 - 2) << HOT_MAXLEVEL; }
            const int s = 1 << (HOT_MAXLEVEL - lev);
            // per-axis gap between the two cubes, squared distance in grid units (< 2^50)
            const uint32_t gx = (uint32_t)max(0, max(cx - ghx, gox - (cx + s)));
            const uint32_t gy = (uint32_t)max(0, max(cy - ghy, goy - (cy + s)));
            const uint32_t gz = (uint32_t)max(0, max(cz - ghz, goz - (cz + s)));
            const unsigned long long d2 = (unsigned long long)gx * gx + (unsigned long long)gy * gy + (unsigned long long)gz * gz;
            bool acc; int ocode = 0, where = 0; // BG: 0 inside K_G, 1 outside, 2 across its boundary
            if (BG && v) {
                const bool out = cx + s <= klx || cx >= khx || cy + s <= kly || cy >= khy || cz + s <= klz || cz >= khz;
                const bool in = cx >= klx && cx + s <= khx && cy >= kly && cy + s <= khy && cz >= klz && cz + s <= khz;
                where = out ? 1 : (in ? 0 : 2);
            }
            if (!TOL) { acc = v && d2 >= P.mac_t[lev] && (!BG || where != 2); if (BG) ocode = where == 1; } // == (double)(s*s) < theta^2 * (double)d2, see mac_table()
            else {
                acc = false;
                if (v) {
                    const CellA A = P.cellA[c];
                    const float4 mb = P.cellMac[c]; // b, 3 B2, 4 sqrt(B2 B4), 6 b B4
                    double zx = A.zx, zy = A.zy, zz = A.zz;
                    if (PER) { zx += (double)(im / 25 - 2) * P.size; zy += (double)((im / 5) % 5 - 2) * P.size; zz += (double)(im % 5 - 2) * P.size; }
                    const double ax = fmax(fabs(zx - gcx) - gh, 0.0), ay = fmax(fabs(zy - gcy) - gh, 0.0), az = fmax(fabs(zz - gcz) - gh, 0.0);
                    const double R2 = ax * ax + ay * ay + az * az, R = sqrt(R2), b = (double)mb.x;
                    if (R > b && R - b > P.hreal) { // (spline softening: every body of the cell beyond the kernel's support)
                        const double t = P.tol * (R - b) * (R - b); // bound_p <= tol  <=>  c_p <= tol (R-b)^2 R^(p+1)
                        if ((double)mb.y <= t * R2) { acc = true; ocode = 0; }
                        else if ((double)mb.z <= t * R2 * R) { acc = true; ocode = 1; }
                        else if ((double)mb.w <= t * R2 * R2 * R) { acc = true; ocode = 2; }
                    }
                }
            }
            const bool self = v && c == gcell && (!PER || im == 62);
            const bool rej_leaf = v && !acc && leaf && !self;
            const bool open = v && !acc && !leaf && !self;
            const uint32_t macc = __ballot_sync(FULL, acc), mopen = __ballot_sync(FULL, open), mrej = __ballot_sync(FULL, rej_leaf);
            // accepted cells -> P-C list
            if (acc) {
                const uint32_t p = npc + __popc(macc & lt);
                // periodic: cells of the coarsest levels are marked; their monopoles are summed in fp64 (hot_periodic.cu)
                if (p < scap) { spc[p] = ((PER && !BG && lev <= HOT_COARSE_LEVEL) ? (c | HOT_COARSE_FLAG) : c) | ((TOL || BG) ? (uint32_t)ocode << HOT_ORDER_SHIFT : 0u); if (PER) ipc[p] = (uint8_t)im; }
            }
            npc += __popc(macc);
            if (TOL || BG) { n0 += __popc(__ballot_sync(FULL, acc && ocode == 0)); n2 += __popc(__ballot_sync(FULL, acc && ocode == 1)); }
            // rejected leaves -> one body run each (a leaf holds <= 32 bodies except at the finest level)
            if (mrej) {
                nbody += rej_leaf ? cnt : 0u; // per lane; summed over the warp when the walk of the group is done
                const bool small = rej_leaf && cnt <= 32u;
                const uint32_t msmall = __ballot_sync(FULL, small);
                uint32_t mbig = mrej & ~msmall;
                if (small) {
                    const uint32_t p = nrun + __popc(msmall & lt);
                    if (p < scap) { spp[p] = wc.z | ((cnt - 1u) << HOT_RUN_SHIFT); if (PER) ipp[p] = (uint8_t)im; }
                }
                nrun += __popc(msmall);
                while (mbig) { // a finest-level leaf with more than 32 bodies: ceil(n/32) runs
                    const int src = __ffs(mbig) - 1;
                    mbig &= mbig - 1;
                    const uint32_t f = __shfl_sync(FULL, wc.z, src), n = __shfl_sync(FULL, cnt, src);
                    const int si = PER ? __shfl_sync(FULL, im, src) : 0;
                    const uint32_t nr = (n + 31u) / 32u;
                    for (uint32_t r = lane; r < nr; r += 32) {
                        const uint32_t p = nrun + r, k = min(32u, n - 32u * r);
                        if (p < scap) { spp[p] = (f + 32u * r) | ((k - 1u) << HOT_RUN_SHIFT); if (PER) ipp[p] = (uint8_t)si; }
                    }
                    nrun += nr;
                }
            }
            // opened cells -> their child run into the ring
            if (open) {
                const int p = (head + top + __popc(mopen & lt)) & M;
                ring[p] = wc.z | ((cnt - 1u) << 28);
                if (PER) rimg[p] = (uint8_t)im;
            }
            top += __popc(mopen);
            if (BG) { // virtual cubes: the cube of a rejected leaf, the empty octants of an opened cell -- outside or across K_G only
                uint32_t miss = 0;
                if (open && where != 0) miss = ~P.cmask[c] & 0xffu;
                const int nv = (rej_leaf && where != 0) ? 1 : __popc(miss);
                int incl = nv;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(FULL, incl, o); if (lane >= o) incl += y; }
                const int tot = __shfl_sync(FULL, incl, 31);
                if (tot) {
                    if ((int64_t)vtop + tot > P.vstack_cap) { if (lane == 0) atomicOr(P.errflag, 16); }
                    else {
                        uint32_t at = vtop + (uint32_t)(incl - nv);
                        const int ux = cx - ((im / 25 - 2) << HOT_MAXLEVEL), uy = cy - (((im / 5) % 5 - 2) << HOT_MAXLEVEL), uz = cz - ((im % 5 - 2) << HOT_MAXLEVEL); // unshifted corner
                        if (rej_leaf && where != 0) vstack[at] = make_uint4((uint32_t)ux | ((uint32_t)uy << 21), ((uint32_t)uy >> 11) | ((uint32_t)uz << 10), (uint32_t)lev, (uint32_t)im);
                        else
                            for (uint32_t mm = miss; mm; mm &= mm - 1) {
                                const int q8 = __ffs((int)mm) - 1, hs = s >> 1;
                                const uint32_t qx = (uint32_t)(ux + ((q8 >> 2) & 1) * hs), qy = (uint32_t)(uy + ((q8 >> 1) & 1) * hs), qz = (uint32_t)(uz + (q8 & 1) * hs);
                                vstack[at++] = make_uint4(qx | (qy << 21), (qy >> 11) | (qz << 10), (uint32_t)lev + 1u, (uint32_t)im);
                            }
                        vtop += (uint32_t)tot;
                    }
                }
            }
            __syncwarp();
        }
        if (BG) { // the virtual cubes: inside K_G dropped; outside accepted by the criterion (or at the finest level); else subdivided
            while (vtop > 0) {
                const uint32_t take = min(32u, vtop);
                vtop -= take;
                __syncwarp();
                uint4 e = make_uint4(0, 0, 0, 0);
                const bool have = (uint32_t)lane < take;
                if (have) e = vstack[vtop + lane];
                const int lev = (int)e.z, im = (int)e.w, s = 1 << (HOT_MAXLEVEL - lev);
                const int ux = (int)(e.x & 0x1fffffu), uy = (int)((e.x >> 21) | ((e.y & 0x3ffu) << 11)), uz = (int)((e.y >> 10) & 0x1fffffu);
                const int cx = ux + ((im / 25 - 2) << HOT_MAXLEVEL), cy = uy + (((im / 5) % 5 - 2) << HOT_MAXLEVEL), cz = uz + ((im % 5 - 2) << HOT_MAXLEVEL);
                const bool out = cx + s <= klx || cx >= khx || cy + s <= kly || cy >= khy || cz + s <= klz || cz >= khz;
                const bool in = cx >= klx && cx + s <= khx && cy >= kly && cy + s <= khy && cz >= klz && cz + s <= khz;
                const uint32_t gx = (uint32_t)max(0, max(cx - ghx, gox - (cx + s)));
                const uint32_t gy = (uint32_t)max(0, max(cy - ghy, goy - (cy + s)));
                const uint32_t gz = (uint32_t)max(0, max(cz - ghz, goz - (cz + s)));
                const unsigned long long d2 = (unsigned long long)gx * gx + (unsigned long long)gy * gy + (unsigned long long)gz * gz;
                const bool accv = have && out && (d2 >= P.mac_t[lev] || lev == HOT_MAXLEVEL);
                const bool sub = have && !in && !accv;
                const uint32_t macc = __ballot_sync(FULL, accv), msub = __ballot_sync(FULL, sub);
                if (accv) { const uint32_t q = npv + __popc(macc & lt); if (q < (uint32_t)P.vstage_cap) vstage[q] = e; }
                npv += __popc(macc);
                if (msub) {
                    const uint32_t tot = 8u * __popc(msub);
                    if ((int64_t)vtop + tot > P.vstack_cap) { if (lane == 0) atomicOr(P.errflag, 16); break; }
                    if (sub) {
                        uint32_t at = vtop + 8u * __popc(msub & lt);
                        const int hs = s >> 1;
                        for (int q8 = 0; q8 < 8; ++q8) {
                            const uint32_t qx = (uint32_t)(ux + ((q8 >> 2) & 1) * hs), qy = (uint32_t)(uy + ((q8 >> 1) & 1) * hs), qz = (uint32_t)(uz + (q8 & 1) * hs);
                            vstack[at++] = make_uint4(qx | (qy << 21), (qy >> 11) | (qz << 10), (uint32_t)lev + 1u, (uint32_t)im);
                        }
                    }
                    vtop += tot;
                }
            }
            if (npv > (uint32_t)P.vstage_cap) { if (lane == 0) atomicOr(P.errflag, 16); continue; }
        }
        nbody = __reduce_add_sync(FULL, nbody);
        // the group's lists are complete: take a slice of the arena and move them there; the body
        // runs are expanded to one body index per entry on the way (32 entries per step)
        if (npc > scap || nrun > scap) { if (lane == 0) atomicOr(P.errflag, 8); continue; }
        unsigned long long pcb = 0, ppb = 0;
        int ok = 1;
        if (lane == 0) {
            pcb = atomicAdd(P.tops, (unsigned long long)npc);
            ppb = atomicAdd(P.tops + 1, (unsigned long long)nbody);
            ok = pcb + npc <= P.cappc && ppb + nbody <= P.cappp;
            if (!ok) atomicMin(P.first_fail, (int)gi);
        }
        ok = __shfl_sync(FULL, ok, 0);
        if (!ok) continue;
        pcb = __shfl_sync(FULL, pcb, 0); ppb = __shfl_sync(FULL, ppb, 0);
        __syncwarp();
        if (!TOL && !BG) {
            // four loads in flight per lane: the staged list comes back from L2, and a one-at-a-time copy loop was 20% of the
            // kernel's warp samples
            for (uint32_t j0 = lane; j0 < npc; j0 += 128) {
                uint32_t v[4]; uint8_t vi[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const uint32_t j = j0 + 32u * k;
                    v[k] = j < npc ? spc[j] : 0u;
                    if (PER) vi[k] = j < npc ? ipc[j] : (uint8_t)0;
                }
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const uint32_t j = j0 + 32u * k;
                    if (j < npc) { P.pclist[pcb + j] = v[k]; if (PER) P.pcimg[pcb + j] = vi[k]; }
                }
            }
        } else { // three stable passes: monopoles, quadrupoles, hexadecapoles; the order bits are dropped
            uint32_t base = 0;
            for (uint32_t o = 0; o < 3; ++o)
                for (uint32_t j0 = 0; j0 < npc; j0 += 32) {
                    const uint32_t j = j0 + lane;
                    const uint32_t e = j < npc ? spc[j] : 0u;
                    const bool hit = j < npc && ((e >> HOT_ORDER_SHIFT) & 3u) == o;
                    const uint32_t m = __ballot_sync(FULL, hit);
                    if (hit) {
                        const uint32_t q = base + __popc(m & lt);
                        P.pclist[pcb + q] = e & ~(3u << HOT_ORDER_SHIFT);
                        if (PER) P.pcimg[pcb + q] = ipc[j];
                    }
                    base += __popc(m);
                }
        }
        {
            // The body runs are expanded through the warp's ring buffer, which is empty now: 32 runs per step, one per lane;
            // an exclusive scan of the run lengths says where each goes; every lane writes its run into the ring (strided
            // shared-memory stores), then the warp copies the ring out coalesced.  (A warp scan per 32 OUTPUT entries, as in
            // round 1, was 19% of the kernel's instructions; writing the runs straight to global memory, one run per lane,
            // was slower still: partial-sector stores.)
            uint32_t out = 0;
            for (uint32_t r = 0; r < nrun;) {
                uint32_t e = 0; int eim = 62, ecnt = 0;
                if (r + lane < nrun) { e = spp[r + lane]; if (PER) eim = ipp[r + lane]; ecnt = (int)(e >> HOT_RUN_SHIFT) + 1; }
                int incl = ecnt;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(FULL, incl, o); if (lane >= o) incl += y; }
                const bool take = ecnt > 0 && incl <= RING; // a run holds <= 32 bodies: at least 16 runs fit
                const int ne = __popc(__ballot_sync(FULL, take));
                const int tot = __shfl_sync(FULL, incl, ne - 1);
                const uint32_t first = e & ((1u << HOT_RUN_SHIFT) - 1u);
                const int at = incl - ecnt;
                const int longest = __reduce_max_sync(FULL, take ? ecnt : 0);
                for (int k = 0; k < longest; ++k)
                    if (take && k < ecnt) { ring[at + k] = first + (uint32_t)k; if (PER) rimg[at + k] = (uint8_t)eim; }
                __syncwarp();
                for (int j = lane; j < tot; j += 32) { P.pplist[ppb + out + j] = ring[j]; if (PER) P.ppimg[ppb + out + j] = rimg[j]; }
                __syncwarp();
                out += (uint32_t)tot; r += (uint32_t)ne;
            }
        }
        if (BG) { // the accepted virtual cubes: their own arena
            unsigned long long pvb = 0;
            if (lane == 0) {
                pvb = atomicAdd(P.tops + 2, (unsigned long long)npv);
                if (pvb + npv > P.cappv) { atomicOr(P.errflag, 32); pvb = ~0ull; }
            }
            pvb = __shfl_sync(FULL, pvb, 0);
            __syncwarp();
            if (pvb != ~0ull) for (uint32_t j = lane; j < npv; j += 32) P.pvlist[pvb + j] = vstage[j];
            if (lane == 0) { P.lpv[gi] = npv; P.pvoff[gi] = pvb == ~0ull ? 0ull : pvb; }
        }
        if (lane == 0) {
            P.lpc[gi] = npc; P.lpp[gi] = nbody; P.lvis[gi] = nvis;
            if (TOL || BG) { P.lpc0[gi] = n0; P.lpc2[gi] = n2; }
            P.pcoff[gi] = pcb; P.ppoff[gi] = ppb;
        }
        __syncwarp();
    }
    if (lane == 0 && WSLOT(uint32_t, SLOT_NSPILL)) atomicAdd(&P.stat[1], (unsigned long long)WSLOT(uint32_t, SLOT_NSPILL));
#undef gi
#undef spc
#undef spp
#undef ipc
#undef ipp
#undef gstack
#undef vstack
#undef vstage
}

int walk_grid_warps() { // resident warps of the walk grid: blocks/SM of the variant that fits fewest
    static int nw = 0;
    if (!nw) {
        int dev = 0, nsm = 0, occ = 1 << 20, o = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, walk_kernel<false, false, false>, WALK_WARPS * 32, 0) == cudaSuccess && o > 0 && o < occ) occ = o;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, walk_kernel<true, false, false>, WALK_WARPS * 32, 0) == cudaSuccess && o > 0 && o < occ) occ = o;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, walk_kernel<false, true, false>, WALK_WARPS * 32, 0) == cudaSuccess && o > 0 && o < occ) occ = o;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, walk_kernel<true, true, false>, WALK_WARPS * 32, 0) == cudaSuccess && o > 0 && o < occ) occ = o;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, walk_kernel<true, false, true>, WALK_WARPS * 32, 0) == cudaSuccess && o > 0 && o < occ) occ = o;
        if (occ == 1 << 20) occ = 1;
        cudaGetLastError();
        nw = nsm * occ * WALK_WARPS;
    }
    return nw;
}
cudaError_t launch_walk(const WalkArgs& a, cudaStream_t st) {
    const int nb = walk_grid_warps() / WALK_WARPS;
    HOT_LAUNCHED(1);
    if (a.tolmode) {
        if (a.periodic) walk_kernel<true, true, false><<<nb, WALK_WARPS * 32, 0, st>>>(a);
        else walk_kernel<false, true, false><<<nb, WALK_WARPS * 32, 0, st>>>(a);
    } else if (a.periodic && a.bgmode) walk_kernel<true, false, true><<<nb, WALK_WARPS * 32, 0, st>>>(a);
    else if (a.periodic) walk_kernel<true, false, false><<<nb, WALK_WARPS * 32, 0, st>>>(a);
    else walk_kernel<false, false, false><<<nb, WALK_WARPS * 32, 0, st>>>(a);
    return cudaGetLastError();
}

// interaction and visit counts of the last walk, summed over the groups
__global__ void __launch_bounds__(256) group_stats_kernel(const GroupRec* __restrict__ group, const uint32_t* __restrict__ lpc,
                                                          const uint32_t* __restrict__ lpp, const uint32_t* __restrict__ lvis,
                                                          const uint32_t* __restrict__ lpc0, const uint32_t* __restrict__ lpc2, int64_t ng,
                                                          unsigned long long* __restrict__ stat) {
    unsigned long long vis = 0, spp = 0, spc = 0, s0 = 0, s2 = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < ng; i += (int64_t)gridDim.x * blockDim.x) {
        const unsigned long long n = group[i].count;
        vis += lvis[i]; spc += n * lpc[i]; spp += n * ((unsigned long long)lpp[i] + n); // L_pp counts the group's own bodies too
        if (lpc0) { s0 += n * lpc0[i]; s2 += n * lpc2[i]; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        vis += __shfl_xor_sync(FULL, vis, o); spp += __shfl_xor_sync(FULL, spp, o); spc += __shfl_xor_sync(FULL, spc, o);
        s0 += __shfl_xor_sync(FULL, s0, o); s2 += __shfl_xor_sync(FULL, s2, o);
    }
    if ((threadIdx.x & 31) == 0) { atomicAdd(&stat[0], vis); atomicAdd(&stat[2], spp); atomicAdd(&stat[3], spc); if (lpc0) { atomicAdd(&stat[4], s0); atomicAdd(&stat[5], s2); } }
}
cudaError_t launch_group_stats(const GroupRec* group, const uint32_t* lpc, const uint32_t* lpp, const uint32_t* lvis,
                               const uint32_t* lpc0, const uint32_t* lpc2, int64_t ng, unsigned long long* stat, cudaStream_t st) {
    HOT_LAUNCHED(1);
    const unsigned nb = (unsigned)((ng + 255) / 256 < 1184 ? (ng + 255) / 256 : 1184);
    group_stats_kernel<<<nb, 256, 0, st>>>(group, lpc, lpp, lvis, lpc0, lpc2, ng, stat);
    return cudaGetLastError();
}

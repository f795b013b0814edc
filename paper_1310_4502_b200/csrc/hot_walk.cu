// hot_walk.cu -- S7: the per-sink-group tree walk that emits the interaction lists.
//
// One warp owns one sink group at a time (persistent grid, dynamic group counter).  The warp
// traverses the tree cooperatively: it pops up to 32 cells from a shared-memory deque, every lane
// applies the multipole acceptance criterion to one cell (integer geometry, one IEEE double multiply
// and compare -- DESIGN.md R-7), and ballots sort the cells into
//   accepted      -> cell index appended to the group's particle-cell list,
//   rejected leaf -> its body indices appended to the group's particle-particle list,
//   else          -> its run of children pushed on the deque.
// The kernel runs twice per hot_forces: a COUNT pass (list lengths per group; an exclusive scan of
// them gives every group a contiguous slice of the list arena) and a FILL pass that writes the lists.
// The walk is latency-bound (dependent 16-byte cell loads), so it runs at high occupancy (few
// registers, ~2.6 KB of shared memory per warp) and leaves the FP32-heavy evaluation to hot_forces.cu.
#include "hot_internal.h"

#define FULL 0xffffffffu
#define WALK_WARPS 8   // warps per block
#define RING 512       // deque entries per warp (runs of <= 8 sibling cells); a power of two

// pending work: ring buffer used as a deque.  An entry is a run of sibling cells
// (first cell | (count-1) << 28, count <= 8): opening a cell pushes ONE entry.  While the ring is short
// the warp pops the OLDEST entries (breadth-first: keeps the frontier wide and the 32 lanes busy);
// once it holds RING/4 entries it pops the NEWEST (depth-first: bounded growth).  If it still fills
// up, the oldest entries spill to a per-warp arena in global memory.
template <bool PER, bool FILL>
__global__ void __launch_bounds__(WALK_WARPS * 32) walk_kernel(const __grid_constant__ WalkArgs P) {
    __shared__ uint32_t s_ring[WALK_WARPS][RING];
    __shared__ uint8_t s_img[PER ? WALK_WARPS : 1][PER ? RING : 1];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t* const ring = s_ring[w];
    uint8_t* const rimg = s_img[PER ? w : 0];
    const int64_t gwarp = (int64_t)blockIdx.x * WALK_WARPS + w;
    uint32_t* const gstack = P.gstack + gwarp * P.gstack_cap * (PER ? 2 : 1);
    const uint32_t lt = (1u << lane) - 1u;
    constexpr int M = RING - 1, DEQ_DFS = RING / 4, NIMG = PER ? 125 : 1;
    const double theta2 = P.theta2;
    unsigned long long nvisit = 0, nspill = 0, sum_pp = 0, sum_pc = 0;

    while (true) {
        unsigned int gi = 0;
        if (lane == 0) gi = atomicAdd(P.counter, 1u);
        gi = __shfl_sync(FULL, gi, 0) + (unsigned int)P.g0;
        if ((int64_t)gi >= P.g1) break;
        const GroupRec g = P.group[gi];
        const uint32_t gcell = g.cell;
        // group cube on the integer grid
        const WalkCell gw = P.wcell[gcell];
        const int gs = 1 << (HOT_MAXLEVEL - (int)(gw.w >> 27));
        const int gox = (int)(gw.x & 0x1fffffu), goy = (int)((gw.x >> 21) | ((gw.y & 0x3ffu) << 11)), goz = (int)((gw.y >> 10) & 0x1fffffu);
        uint32_t* pcl = nullptr; uint32_t* ppl = nullptr; uint8_t* pci = nullptr; uint8_t* ppi = nullptr;
        if (FILL) {
            const uint64_t pb = P.pcoff[gi] - P.pcbase, bb = P.ppoff[gi] - P.ppbase;
            pcl = P.pclist + pb; ppl = P.pplist + bb;
            if (PER) { pci = P.pcimg + pb; ppi = P.ppimg + bb; }
        }
        uint32_t npc = 0, npp = 0; // list lengths so far
        int head = 0, top = 0, gtop = 0, next_img = 0;
        while (true) {
            if (top == 0) {
                if (gtop > 0) { // refill from the global arena
                    const int mv = gtop > RING / 2 ? RING / 2 : gtop;
                    for (int t = lane; t < mv; t += 32) {
                        ring[(head + t) & M] = gstack[gtop - mv + t];
                        if (PER) rimg[(head + t) & M] = (uint8_t)gstack[P.gstack_cap + gtop - mv + t];
                    }
                    gtop -= mv; top = mv;
                } else if (next_img < NIMG) { // seed: the root once per image (lane = image)
                    const int im = next_img + lane;
                    if (im < NIMG) { ring[(head + lane) & M] = 0u; if (PER) rimg[(head + lane) & M] = (uint8_t)im; }
                    top = min(32, NIMG - next_img);
                    next_img += top;
                } else break;
                __syncwarp();
            }
            if (RING - top < 32) { // no room for 32 pushes: spill the oldest entries, keep 128 on chip
                const int keep = 128, mv = top - keep;
                if ((int64_t)gtop + mv > P.gstack_cap) { if (lane == 0) atomicOr(P.errflag, 4); break; }
                for (int t = lane; t < mv; t += 32) {
                    gstack[gtop + t] = ring[(head + t) & M];
                    if (PER) gstack[P.gstack_cap + gtop + t] = rimg[(head + t) & M]; // image ids: second half of the arena
                }
                __syncwarp();
                gtop += mv; head = (head + mv) & M; top = keep; ++nspill;
            }
            // take whole entries while they hold <= 32 cells in total, one cell per lane
            uint32_t c; int im = PER ? 62 : 0, nt;
            {
                const bool dfs = top >= DEQ_DFS;
                const int at = dfs ? (head + top - 1 - lane) & M : (head + lane) & M;
                uint32_t e = 0; int eim = 62, ecnt = 0;
                if (lane < top) { e = ring[at]; if (PER) eim = rimg[at]; ecnt = (int)(e >> 28) + 1; }
                int incl = ecnt;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(FULL, incl, o); if (lane >= o) incl += y; }
                const bool take = lane < top && incl <= 32;
                const int ne = __popc(__ballot_sync(FULL, take)); // >= 1: an entry holds <= 8 cells
                nt = __shfl_sync(FULL, incl, ne - 1);
                const int excl = incl - ecnt;
                const uint32_t starts = __reduce_or_sync(FULL, take ? (1u << excl) : 0u);
                const int src = max(0, __popc(starts & ((2u << lane) - 1u)) - 1); // entry that holds this lane's cell
                const uint32_t eb = __shfl_sync(FULL, e & 0x0fffffffu, src);
                const int ex = __shfl_sync(FULL, excl, src);
                if (PER) im = __shfl_sync(FULL, eim, src);
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
            const uint32_t macc = __ballot_sync(FULL, acc), mopen = __ballot_sync(FULL, open);
            uint32_t mrej = __ballot_sync(FULL, rej_leaf);
            // accepted cells -> P-C list
            if (FILL && acc) { const uint32_t p = npc + __popc(macc & lt); pcl[p] = c; if (PER) pci[p] = (uint8_t)im; }
            npc += __popc(macc);
            // rejected leaves -> their bodies to the P-P list
            if (mrej) {
                if (FILL) {
                    while (mrej) {
                        const int src = __ffs(mrej) - 1;
                        mrej &= mrej - 1;
                        const uint32_t f = __shfl_sync(FULL, wc.z, src), n = __shfl_sync(FULL, cnt, src);
                        const int si = PER ? __shfl_sync(FULL, im, src) : 0;
                        for (uint32_t j = lane; j < n; j += 32) { ppl[npp + j] = f + j; if (PER) ppi[npp + j] = (uint8_t)si; }
                        npp += n;
                    }
                } else {
                    uint32_t nb = rej_leaf ? cnt : 0u;
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) nb += __shfl_xor_sync(FULL, nb, o);
                    npp += nb;
                }
            }
            // opened cells -> their child run into the ring
            if (open) {
                const int p = (head + top + __popc(mopen & lt)) & M;
                ring[p] = wc.z | ((cnt - 1u) << 28);
                if (PER) rimg[p] = (uint8_t)im;
            }
            top += __popc(mopen);
            __syncwarp();
        }
        if (!FILL && lane == 0) {
            P.lpc[gi] = npc; P.lpp[gi] = npp;
            // interaction counts: every sink of the group against the lists; L_pp counts the group's own bodies too
            sum_pc += (unsigned long long)g.count * npc; sum_pp += (unsigned long long)g.count * ((unsigned long long)npp + g.count);
        }
    }
    if (lane == 0 && !FILL) {
        atomicAdd(&P.stat[0], nvisit); atomicAdd(&P.stat[1], nspill);
        atomicAdd(&P.stat[2], sum_pp); atomicAdd(&P.stat[3], sum_pc);
    }
}

int walk_grid_warps() { // resident warps of the walk grid: blocks/SM of the variant that fits fewest
    static int nw = 0;
    if (!nw) {
        int dev = 0, nsm = 0, occ = 0, o = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
        occ = 1 << 20;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, walk_kernel<false, false>, WALK_WARPS * 32, 0) == cudaSuccess && o > 0 && o < occ) occ = o;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, walk_kernel<false, true>, WALK_WARPS * 32, 0) == cudaSuccess && o > 0 && o < occ) occ = o;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, walk_kernel<true, false>, WALK_WARPS * 32, 0) == cudaSuccess && o > 0 && o < occ) occ = o;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, walk_kernel<true, true>, WALK_WARPS * 32, 0) == cudaSuccess && o > 0 && o < occ) occ = o;
        if (occ == 1 << 20) occ = 1;
        cudaGetLastError();
        nw = nsm * occ * WALK_WARPS;
    }
    return nw;
}
cudaError_t launch_walk(const WalkArgs& a, bool fill, cudaStream_t st) {
    const int nb = walk_grid_warps() / WALK_WARPS;
    HOT_LAUNCHED(1);
    if (a.periodic) {
        if (fill) walk_kernel<true, true><<<nb, WALK_WARPS * 32, 0, st>>>(a);
        else walk_kernel<true, false><<<nb, WALK_WARPS * 32, 0, st>>>(a);
    } else {
        if (fill) walk_kernel<false, true><<<nb, WALK_WARPS * 32, 0, st>>>(a);
        else walk_kernel<false, false><<<nb, WALK_WARPS * 32, 0, st>>>(a);
    }
    return cudaGetLastError();
}

// ---- exclusive scan of the per-group list lengths into 64-bit offsets ----------------------------
// off[i] = sum_{j<i} len[j], off[n] = total.  Three kernels: per-block sums, scan of the block sums
// (one block), per-block exclusive scan + block offset.
#define SCAN_THREADS 256
#define SCAN_ITEMS 8
#define SCAN_TILE (SCAN_THREADS * SCAN_ITEMS)
__device__ __forceinline__ unsigned long long block_excl_scan(unsigned long long v, unsigned long long* wsum, unsigned long long& total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    unsigned long long x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { unsigned long long y = __shfl_up_sync(FULL, x, o); if (lane >= o) x += y; }
    if (lane == 31) wsum[w] = x;
    __syncthreads();
    if (w == 0) {
        unsigned long long s = lane < SCAN_THREADS / 32 ? wsum[lane] : 0ull, t = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { unsigned long long y = __shfl_up_sync(FULL, t, o); if (lane >= o) t += y; }
        if (lane < SCAN_THREADS / 32) wsum[lane] = t - s;
        if (lane == 31) wsum[SCAN_THREADS / 32] = t;
    }
    __syncthreads();
    total = wsum[SCAN_THREADS / 32];
    const unsigned long long r = wsum[w] + x - v;
    __syncthreads();
    return r;
}
__global__ void __launch_bounds__(SCAN_THREADS) scan_tile_sums(const uint32_t* __restrict__ len, int64_t n, unsigned long long* __restrict__ tsum) {
    __shared__ unsigned long long wsum[SCAN_THREADS / 32 + 1];
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    unsigned long long v = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) if (base + k < n) v += len[base + k];
    unsigned long long total;
    block_excl_scan(v, wsum, total);
    if (threadIdx.x == 0) tsum[blockIdx.x] = total;
}
__global__ void __launch_bounds__(SCAN_THREADS) scan_tile_offsets(unsigned long long* __restrict__ tsum, int64_t ntiles) {
    __shared__ unsigned long long wsum[SCAN_THREADS / 32 + 1];
    __shared__ unsigned long long carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int64_t b0 = 0; b0 < ntiles; b0 += SCAN_THREADS) {
        const int64_t i = b0 + threadIdx.x;
        const unsigned long long v = i < ntiles ? tsum[i] : 0ull;
        unsigned long long total;
        const unsigned long long e = block_excl_scan(v, wsum, total);
        const unsigned long long c = carry;
        if (i < ntiles) tsum[i] = c + e;
        __syncthreads();
        if (threadIdx.x == 0) carry = c + total;
        __syncthreads();
    }
    if (threadIdx.x == 0) tsum[ntiles] = carry;
}
__global__ void __launch_bounds__(SCAN_THREADS) scan_apply(const uint32_t* __restrict__ len, int64_t n, const unsigned long long* __restrict__ tsum,
                                                           int64_t ntiles, unsigned long long* __restrict__ off) {
    __shared__ unsigned long long wsum[SCAN_THREADS / 32 + 1];
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    uint32_t l[SCAN_ITEMS];
    unsigned long long v = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) { l[k] = base + k < n ? len[base + k] : 0u; v += l[k]; }
    unsigned long long total;
    unsigned long long run = tsum[blockIdx.x] + block_excl_scan(v, wsum, total);
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) { if (base + k < n) off[base + k] = run; run += l[k]; }
    if (blockIdx.x == 0 && threadIdx.x == 0) off[n] = tsum[ntiles];
}
size_t scan_scratch_elems(int64_t n) { return (size_t)((n + SCAN_TILE - 1) / SCAN_TILE) + 1; }
cudaError_t launch_scan_u32_to_u64(const uint32_t* len, int64_t n, unsigned long long* scratch, unsigned long long* off, cudaStream_t st) {
    const int64_t nt = (n + SCAN_TILE - 1) / SCAN_TILE;
    HOT_LAUNCHED(3);
    scan_tile_sums<<<(unsigned)nt, SCAN_THREADS, 0, st>>>(len, n, scratch);
    scan_tile_offsets<<<1, SCAN_THREADS, 0, st>>>(scratch, nt);
    scan_apply<<<(unsigned)nt, SCAN_THREADS, 0, st>>>(len, n, scratch, nt, off);
    return cudaGetLastError();
}

// chunk boundaries: bounds[0] = 0, bounds[k+1] = largest g with (pcoff[g]-pcoff[bounds[k]] <= cappc and
// ppoff[g]-ppoff[bounds[k]] <= cappp); *nchunks = number of chunks, or -1 if one group alone does not fit.
__global__ void chunk_bounds_kernel(const unsigned long long* __restrict__ pcoff, const unsigned long long* __restrict__ ppoff, int64_t ng,
                                    unsigned long long cappc, unsigned long long cappp, int64_t* __restrict__ bounds, int maxchunks,
                                    int* __restrict__ nchunks) {
    int k = 0;
    int64_t g0 = 0;
    bounds[0] = 0;
    while (g0 < ng) {
        int64_t lo = g0, hi = ng; // largest g in (g0, ng] that fits
        while (hi - lo > 0) {
            const int64_t mid = (lo + hi + 1) >> 1;
            if (pcoff[mid] - pcoff[g0] <= cappc && ppoff[mid] - ppoff[g0] <= cappp) lo = mid; else hi = mid - 1;
        }
        if (lo == g0 || k + 1 >= maxchunks) { *nchunks = -1; return; }
        bounds[++k] = lo;
        g0 = lo;
    }
    *nchunks = k;
}
cudaError_t launch_chunk_bounds(const unsigned long long* pcoff, const unsigned long long* ppoff, int64_t ng, unsigned long long cappc,
                                unsigned long long cappp, int64_t* bounds, int maxchunks, int* nchunks, cudaStream_t st) {
    HOT_LAUNCHED(1);
    chunk_bounds_kernel<<<1, 1, 0, st>>>(pcoff, ppoff, ng, cappc, cappp, bounds, maxchunks, nchunks);
    return cudaGetLastError();
}

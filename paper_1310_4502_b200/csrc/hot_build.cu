// hot_build.cu -- S1 keygen, S2 radix sort, S3 gather, S4 tree + hash, S5 sink groups.
// All stages are HBM-bound streaming kernels; see DESIGN.md "Kernels" for bytes per particle.
#include "hot_internal.h"

#define FULL 0xffffffffu

// ------------------------------------------------------------------------------------------
// S1 keys.  PAPER.md:150 defers the coordinate -> key mapping to WS93; reading (R-1):
// t = fl32(fl32(x - lo) * fl32(1/size)), i = floor(t * 2^21), 63-bit Morton interleave with x the
// most significant bit of each triple, placeholder bit 63.  The subtract and the multiply are
// separate IEEE fp32 operations (no FMA contraction): they define the key.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint64_t spread21(uint32_t v) {
    uint64_t x = v & 0x1fffffu;
    x = (x | x << 32) & 0x001f00000000ffffull;
    x = (x | x << 16) & 0x001f0000ff0000ffull;
    x = (x | x << 8) & 0x100f00f00f00f00full;
    x = (x | x << 4) & 0x10c30c30c30c30c3ull;
    x = (x | x << 2) & 0x1249249249249249ull;
    return x;
}
__device__ __forceinline__ uint32_t compact21(uint64_t x) {
    x &= 0x1249249249249249ull;
    x = (x | x >> 2) & 0x10c30c30c30c30c3ull;
    x = (x | x >> 4) & 0x100f00f00f00f00full;
    x = (x | x >> 8) & 0x001f0000ff0000ffull;
    x = (x | x >> 16) & 0x001f00000000ffffull;
    x = (x | x >> 32) & 0x1fffffull;
    return (uint32_t)x;
}
__device__ __forceinline__ uint32_t grid_coord(float x, float lo, float inv, bool& bad) {
    float t = __fmul_rn(__fsub_rn(x, lo), inv);
    if (!(t >= 0.0f) || !(t < 1.0f)) bad = true;
    int i = (int)floorf(__fmul_rn(t, 2097152.0f));
    i = max(0, min(2097151, i));
    return (uint32_t)i;
}
__device__ __forceinline__ uint64_t body_key(float x, float y, float z, float lox, float loy, float loz,
                                             float inv, bool& bad) {
    uint32_t ix = grid_coord(x, lox, inv, bad), iy = grid_coord(y, loy, inv, bad), iz = grid_coord(z, loz, inv, bad);
    return (1ull << 63) | (spread21(ix) << 2) | (spread21(iy) << 1) | spread21(iz);
}
// 4 bodies per thread and trip: three 128-bit loads, two 128-bit key stores (the sort's first pass takes the index from
// the position).  Also writes the bodies as aligned float4 (x,y,z,m) in the caller's order: the gather after the sort
// then fetches one 32-byte sector per body instead of the 3-4 sectors of the separate pos / mass arrays.
// The sort's eight digit histograms are counted here as well (shared-memory atomics, added to `ghist` at the end of
// the block's grid-stride loop): the kernel is HBM-bound, the shared-memory pipe is free.
static cudaError_t sort_clear_scratch(uint32_t* hist, int64_t n, cudaStream_t st);
__device__ __forceinline__ void key_digits(uint32_t (*h)[256], uint64_t k) {
    const uint32_t lo = (uint32_t)k, hi = (uint32_t)(k >> 32);
#pragma unroll
    for (int p = 0; p < 4; ++p) {
        atomicAdd(&h[p][__byte_perm(lo, 0u, 0x4440u + p)], 1u);
        atomicAdd(&h[4 + p][__byte_perm(hi, 0u, 0x4440u + p)], 1u);
    }
}
__global__ void __launch_bounds__(256) keygen_kernel(const float* __restrict__ pos, const float* __restrict__ mass, int64_t n, float lox,
                                                     float loy, float loz, float inv, uint64_t* __restrict__ key,
                                                     float4* __restrict__ bin, uint32_t* __restrict__ ghist, int* __restrict__ errflag, int vec) {
    __shared__ uint32_t h[8][256];
#pragma unroll
    for (int p = 0; p < 8; ++p) h[p][threadIdx.x] = 0;
    __syncthreads();
    bool bad = false;
    const int64_t quads = (n + 3) / 4;
    for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < quads; q += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i0 = q * 4;
        if (vec && i0 + 4 <= n) {
            const float4* p4 = reinterpret_cast<const float4*>(pos) + q * 3;
            float4 a = __ldg(p4), b = __ldg(p4 + 1), c = __ldg(p4 + 2);
            const float4 m = __ldg(reinterpret_cast<const float4*>(mass) + q);
            uint64_t k0 = body_key(a.x, a.y, a.z, lox, loy, loz, inv, bad);
            uint64_t k1 = body_key(a.w, b.x, b.y, lox, loy, loz, inv, bad);
            uint64_t k2 = body_key(b.z, b.w, c.x, lox, loy, loz, inv, bad);
            uint64_t k3 = body_key(c.y, c.z, c.w, lox, loy, loz, inv, bad);
            ulonglong2* ko = reinterpret_cast<ulonglong2*>(key + i0);
            ko[0] = make_ulonglong2(k0, k1);
            ko[1] = make_ulonglong2(k2, k3);
            bin[i0] = make_float4(a.x, a.y, a.z, m.x);
            bin[i0 + 1] = make_float4(a.w, b.x, b.y, m.y);
            bin[i0 + 2] = make_float4(b.z, b.w, c.x, m.z);
            bin[i0 + 3] = make_float4(c.y, c.z, c.w, m.w);
            key_digits(h, k0); key_digits(h, k1); key_digits(h, k2); key_digits(h, k3);
        } else {
            for (int64_t i = i0; i < n && i < i0 + 4; ++i) {
                const uint64_t k = body_key(pos[3 * i], pos[3 * i + 1], pos[3 * i + 2], lox, loy, loz, inv, bad);
                key[i] = k;
                bin[i] = make_float4(pos[3 * i], pos[3 * i + 1], pos[3 * i + 2], mass[i]);
                key_digits(h, k);
            }
        }
    }
    if (bad) atomicOr(errflag, 1);
    __syncthreads();
#pragma unroll
    for (int p = 0; p < 8; ++p) { const uint32_t c = h[p][threadIdx.x]; if (c) atomicAdd(&ghist[p * 256 + threadIdx.x], c); }
}
// `hist` is the sort's scratch (sort_hist_elems(n) words): cleared here, its first 2048 words receive the digit counts
cudaError_t launch_keygen(const float* pos, const float* mass, int64_t n, float lox, float loy, float loz, float inv,
                          uint64_t* key, float4* bin, uint32_t* hist, int* errflag, cudaStream_t st) {
    cudaError_t e = sort_clear_scratch(hist, n, st);
    if (e != cudaSuccess) return e;
    int64_t quads = (n + 3) / 4;
    int64_t blocks = (quads + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    int vec = ((reinterpret_cast<uintptr_t>(pos) | reinterpret_cast<uintptr_t>(mass)) & 15u) == 0; // 128-bit loads need 16-byte aligned bases
    HOT_LAUNCHED(1);
    keygen_kernel<<<(unsigned)blocks, 256, 0, st>>>(pos, mass, n, lox, loy, loz, inv, key, bin, hist, errflag, vec);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// S2 LSD radix sort of (key, idx), 8-bit digits, 8 passes (PAPER.md:150 names an American-flag
// radix sort for the on-node sort; a stable LSD sort gives the unique stable permutation).
// keygen_kernel counts all eight digits of every key (2048 counters); each pass is then ONE kernel: a tile
// (256 threads x 16 keys, held warp-striped so the in-tile order is (warp, round, lane)) ranks its keys,
// publishes its digit counts, lays the tile out in digit order in shared memory, finds the counts of all earlier
// tiles by decoupled look-back and scatters.  The kernel is bound by the shared-memory / LSU data pipe (ncu:
// l1tex__data_pipe_lsu_wavefronts 75% of peak, 51 wavefronts per 32 keys), so its design minimises
// shared-memory operations per key, not instructions.
// Scratch (u32): [0,2048) digit counts, [2048,4096) their exclusive scans, [4096,4104) tile tickets,
// then two look-back state arrays of 256 words per tile (a pass uses one and clears the other).
// ------------------------------------------------------------------------------------------
#define SORT_THREADS 256
#define SORT_ITEMS 16
#define SORT_TILE (SORT_THREADS * SORT_ITEMS)
#define SORT_WARPS (SORT_THREADS / 32)
#define SORT_STATE0 4352
#define SORT_AGG 0x40000000u     // look-back word: the tile's own count of the digit
#define SORT_PREFIX 0x80000000u  //                 the count of the digit in this and all earlier tiles
#define SORT_VALUE 0x3fffffffu

static inline int64_t sort_blocks(int64_t n) { return (n + SORT_TILE - 1) / SORT_TILE; }
size_t sort_hist_elems(int64_t n) { return (size_t)SORT_STATE0 + 2 * (size_t)256 * (size_t)sort_blocks(n); }

// exclusive scan of each of the eight 256-bin histograms; one block of 256 threads
__global__ void __launch_bounds__(256) sort_scan8_kernel(const uint32_t* __restrict__ ghist, uint32_t* __restrict__ dbase) {
    __shared__ uint32_t wtot[8];
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    for (int p = 0; p < 8; ++p) {
        uint32_t v = ghist[p * 256 + tid], x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(FULL, x, o); if (lane >= o) x += y; }
        if (lane == 31) wtot[w] = x;
        __syncthreads();
        uint32_t off = 0;
        for (int j = 0; j < w; ++j) off += wtot[j];
        dbase[p * 256 + tid] = off + x - v;
        __syncthreads();
    }
}
__device__ __forceinline__ uint32_t ld_relaxed(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed(uint32_t* p, uint32_t v) { asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory"); }
// in-place exclusive scan of each row (one block per row); totals[row] = row sum
__global__ void __launch_bounds__(1024) scan_rows_kernel(uint32_t* __restrict__ data, int64_t rowlen, uint32_t* __restrict__ totals) {
    __shared__ uint32_t wsum[32];
    __shared__ uint32_t carry, ctot;
    uint32_t* row = data + (int64_t)blockIdx.x * rowlen;
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int64_t base = 0; base < rowlen; base += 1024) {
        int64_t i = base + threadIdx.x;
        uint32_t v = i < rowlen ? row[i] : 0, x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(FULL, x, o); if (lane >= o) x += y; }
        if (lane == 31) wsum[w] = x;
        __syncthreads();
        if (w == 0) {
            uint32_t s = wsum[lane], t = s;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(FULL, t, o); if (lane >= o) t += y; }
            wsum[lane] = t - s; // exclusive warp offsets
            if (lane == 31) ctot = t;
        }
        __syncthreads();
        uint32_t c = carry;
        if (i < rowlen) row[i] = c + wsum[w] + x - v;
        __syncthreads();
        if (threadIdx.x == 0) carry = c + ctot;
        __syncthreads();
    }
    if (threadIdx.x == 0) totals[blockIdx.x] = carry;
}
// Stable scatter of one tile.  PASS is a template parameter so that a digit is one byte of one key half (PRMT);
// FULLT marks a full tile (every tile but the last): no per-key bounds predicates.
// Shared memory: the digit-ordered tile (keys 32 KB + values 16 KB, dynamic) and 10.5 KB of counters.
#define SORT_MINBLK 3  // resident tiles per SM (tile-size sweep in DESIGN.md)
#define SORT_LOOK 4    // earlier tiles read per look-back round trip
#define SORT_SMEM_BYTES (SORT_TILE * 12)
template <int PASS> __device__ __forceinline__ uint32_t sort_digit(uint64_t k) {
    const uint32_t h = PASS < 4 ? (uint32_t)k : (uint32_t)(k >> 32);
    return __byte_perm(h, 0u, 0x4440u + (PASS & 3));
}
struct SortShared {
    uint32_t wcount[SORT_WARPS][256]; // per warp and digit: keys ranked so far; later the warp's start inside the tile
    uint32_t gbase[256];              // global position of the tile's first key of each digit, minus its local start
    uint32_t wtot[SORT_WARPS];
    uint32_t tile;
};
template <int PASS, bool FULLT>
__device__ __forceinline__ void sort_scatter_tile(SortShared& sh, uint64_t* __restrict__ skey, uint32_t* __restrict__ wmbase,
                                                  const int64_t tile, const int cnt,
                                                  const uint64_t* __restrict__ kin, const uint32_t* __restrict__ vin,
                                                  uint64_t* __restrict__ kout, uint32_t* __restrict__ vout,
                                                  const uint32_t* __restrict__ dbase, uint32_t* __restrict__ state,
                                                  uint32_t* __restrict__ state_next) {
    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    uint32_t* const sval = reinterpret_cast<uint32_t*>(skey + SORT_TILE);
    // two per-warp lane-mask arrays, used by alternate ranking rounds; the tile space is free until the ranks are known
    uint32_t* const wm0 = wmbase + w * 256;
    uint32_t* const wm1 = wm0 + SORT_WARPS * 256;
    uint32_t* const wc = sh.wcount[w];
    const int64_t t0 = tile * SORT_TILE;
    const int l0 = w * (32 * SORT_ITEMS) + lane; // this thread's keys: tile positions l0 + 32 k
    const uint64_t* const kt = kin + t0 + l0;
    uint64_t kk[SORT_ITEMS];
    uint32_t rk[SORT_ITEMS]; // rank among the warp's keys of the same digit, later the position in the digit-ordered tile
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) kk[k] = (FULLT || l0 + 32 * k < cnt) ? __ldg(kt + 32 * k) : ~0ull; // all loads first
    // Rank inside the warp's 16 x 32 keys.  The lanes holding the same digit find each other through a
    // shared-memory atomicOr on a per-warp, per-digit lane mask (MATCH.ANY issues once per 64 clocks per SM
    // on sm_100a -- 115 us of a pass at 2^24 keys; eight ballots per key are no faster than the mask).  Round k
    // uses mask array k & 1: its leader clears the word after the round's reads (second warp barrier), and the next
    // atomicOr on that array is two rounds later; the lowest lane of a digit adds the lanes' number to the warp's
    // count of the digit with one atomicAdd and hands the old count to the others by a shuffle.
    const uint32_t lanebit = 1u << lane, below = lanebit - 1u;
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) {
        const bool valid = FULLT || l0 + 32 * k < cnt;
        const uint32_t d = sort_digit<PASS>(kk[k]);
        uint32_t* const mp = ((k & 1) ? wm1 : wm0) + d;
        if (valid) atomicOr(mp, lanebit);
        __syncwarp();
        const uint32_t m = valid ? *mp : 0u;
        const uint32_t r = __popc(m & below);
        uint32_t old = 0;
        if (valid && r == 0) old = atomicAdd(&wc[d], (uint32_t)__popc(m)); // the lowest lane of the digit counts for all
        old = __shfl_sync(FULL, old, (__ffs((int)m) - 1) & 31);
        __syncwarp(); // every lane has read the mask
        if (valid && r == 0) *mp = 0u;
        rk[k] = old + r;
    }
    __syncthreads();
    // The tile's count of digit tid (the column sum of the warps' counts) is published now; the counts of the earlier
    // tiles are looked up after the tile has been laid out in digit order, when most of them have been published.
    uint32_t mine = 0;
#pragma unroll
    for (int j = 0; j < SORT_WARPS; ++j) mine += sh.wcount[j][tid];
    uint32_t* const mystate = state + tile * 256 + tid;
    st_relaxed(mystate, mine | (tile == 0 ? SORT_PREFIX : SORT_AGG));
    state_next[tile * 256 + tid] = 0u; // the next pass looks back through the other array
    uint32_t off; // start of digit tid in the tile (exclusive scan of the counts)
    {
        uint32_t x = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(FULL, x, o); if (lane >= o) x += y; }
        if (lane == 31) sh.wtot[w] = x;
        __syncthreads();
        off = x - mine;
#pragma unroll
        for (int j = 0; j < SORT_WARPS; ++j) off += j < w ? sh.wtot[j] : 0u;
        uint32_t run = off; // ... and of every warp's keys inside the digit
#pragma unroll
        for (int j = 0; j < SORT_WARPS; ++j) { const uint32_t t = sh.wcount[j][tid]; sh.wcount[j][tid] = run; run += t; }
        __syncthreads();
    }
    // digit-ordered tile in shared memory: keys ...
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) {
        rk[k] += wc[sort_digit<PASS>(kk[k])]; // now: position in the tile
        if (FULLT || l0 + 32 * k < cnt) skey[rk[k]] = kk[k];
    }
    // The values are fetched now and arrive while the keys leave (pass 0: the index is the key's position).
    uint32_t vv[SORT_ITEMS];
    if (PASS == 0) {
#pragma unroll
        for (int k = 0; k < SORT_ITEMS; ++k) vv[k] = (uint32_t)(t0 + l0) + 32u * k;
    } else {
        const uint32_t* const vt = vin + t0 + l0;
#pragma unroll
        for (int k = 0; k < SORT_ITEMS; ++k) vv[k] = (FULLT || l0 + 32 * k < cnt) ? __ldg(vt + 32 * k) : 0u;
    }
    {
        uint32_t excl = 0; // keys with digit tid in earlier tiles
        if (tile != 0) {
            // SORT_LOOK earlier tiles per round trip; an unpublished word is read again after a short sleep
            const uint32_t* q = mystate - 256;
            int64_t left = tile; // earlier tiles not yet added
            bool done = false;
            while (!done) {
                uint32_t v[SORT_LOOK];
#pragma unroll
                for (int j = 0; j < SORT_LOOK; ++j) v[j] = j < left ? ld_relaxed(q - j * 256) : SORT_PREFIX;
                int used = 0;
#pragma unroll
                for (int j = 0; j < SORT_LOOK; ++j) {
                    const bool ok = !done && used == j && (v[j] & (SORT_AGG | SORT_PREFIX)) != 0u;
                    if (ok) { excl += v[j] & SORT_VALUE; ++used; done = (v[j] & SORT_PREFIX) != 0u; }
                }
                q -= used * 256; left -= used;
                if (used == 0) __nanosleep(40);
            }
            st_relaxed(mystate, (excl + mine) | SORT_PREFIX);
        }
        sh.gbase[tid] = dbase[tid] + excl - off; // where the tile's run of this digit goes, minus its place in the tile
    }
    __syncthreads();
    uint32_t gb[SORT_ITEMS]; // destination of tile position p = k * 256 + tid, for the key and then the value
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) {
        const int p = k * SORT_THREADS + tid;
        if (FULLT || p < cnt) {
            const uint64_t key = skey[p];
            gb[k] = sh.gbase[sort_digit<PASS>(key)] + (uint32_t)p;
            kout[gb[k]] = key;
        }
    }
    // ... then the values (their own space: no barrier between)
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k)
        if (FULLT || l0 + 32 * k < cnt) sval[rk[k]] = vv[k];
    __syncthreads();
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) {
        const int p = k * SORT_THREADS + tid;
        if (FULLT || p < cnt) vout[gb[k]] = sval[p];
    }
}
template <int PASS>
__global__ void __launch_bounds__(SORT_THREADS, SORT_MINBLK) sort_scatter_kernel(const uint64_t* __restrict__ kin, const uint32_t* __restrict__ vin,
                                                                    uint64_t* __restrict__ kout, uint32_t* __restrict__ vout, int64_t n,
                                                                    const uint32_t* __restrict__ dbase, uint32_t* __restrict__ ticket,
                                                                    uint32_t* __restrict__ state, uint32_t* __restrict__ state_next) {
    __shared__ SortShared sh;
    extern __shared__ __align__(16) uint64_t sort_tile_space[];
    const int tid = threadIdx.x;
    uint32_t* const z = reinterpret_cast<uint32_t*>(sort_tile_space); // both mask arrays
#pragma unroll
    for (int j = 0; j < SORT_WARPS; ++j) { sh.wcount[j][tid] = 0; z[j * 256 + tid] = 0; z[(SORT_WARPS + j) * 256 + tid] = 0; }
    if (tid == 0) sh.tile = atomicAdd(ticket, 1u); // tiles are taken in launch order: every earlier tile is running or done
    __syncthreads();
    const int64_t tile = sh.tile;
    const int64_t left = n - tile * SORT_TILE;
    if (left >= SORT_TILE) sort_scatter_tile<PASS, true>(sh, sort_tile_space, z, tile, SORT_TILE, kin, vin, kout, vout, dbase, state, state_next);
    else sort_scatter_tile<PASS, false>(sh, sort_tile_space, z, tile, (int)left, kin, vin, kout, vout, dbase, state, state_next);
}
template <int PASS>
static cudaError_t launch_sort_pass(uint64_t* key[2], uint32_t* idx[2], int cur, int64_t n, int64_t nblk, uint32_t* dbase, uint32_t* ticket,
                                    uint32_t* const state[2], cudaStream_t st) {
    static bool attr_set = false; // the 48 KB tile is dynamic shared memory above the default limit
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(sort_scatter_kernel<PASS>, cudaFuncAttributeMaxDynamicSharedMemorySize, SORT_SMEM_BYTES);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    HOT_LAUNCHED(1);
    sort_scatter_kernel<PASS><<<(unsigned)nblk, SORT_THREADS, SORT_SMEM_BYTES, st>>>(key[cur], idx[cur], key[cur ^ 1], idx[cur ^ 1], n, dbase + PASS * 256,
                                                                                     ticket + PASS, state[PASS & 1], state[(PASS & 1) ^ 1]);
    return cudaGetLastError();
}
// digit counters, tile tickets and the first look-back array start at zero
static cudaError_t sort_clear_scratch(uint32_t* hist, int64_t n, cudaStream_t st) {
    return cudaMemsetAsync(hist, 0, ((size_t)SORT_STATE0 + (size_t)256 * sort_blocks(n)) * sizeof(uint32_t), st);
}
cudaError_t launch_radix_sort(uint64_t* key[2], uint32_t* idx[2], int64_t n, uint32_t* hist, cudaStream_t st) {
    const int64_t nblk = sort_blocks(n);
    uint32_t* const ghist = hist;
    uint32_t* const dbase = hist + 2048;
    uint32_t* const ticket = hist + 4096;
    uint32_t* const state[2] = {hist + SORT_STATE0, hist + SORT_STATE0 + (size_t)256 * nblk};
    cudaError_t e;
    HOT_LAUNCHED(1);
    sort_scan8_kernel<<<1, 256, 0, st>>>(ghist, dbase);
    // 8 passes: the result is back in buffer 0.  Pass 0 takes the index from the key's position (idx[0] is not read).
    if ((e = launch_sort_pass<0>(key, idx, 0, n, nblk, dbase, ticket, state, st)) != cudaSuccess) return e;
    if ((e = launch_sort_pass<1>(key, idx, 1, n, nblk, dbase, ticket, state, st)) != cudaSuccess) return e;
    if ((e = launch_sort_pass<2>(key, idx, 0, n, nblk, dbase, ticket, state, st)) != cudaSuccess) return e;
    if ((e = launch_sort_pass<3>(key, idx, 1, n, nblk, dbase, ticket, state, st)) != cudaSuccess) return e;
    if ((e = launch_sort_pass<4>(key, idx, 0, n, nblk, dbase, ticket, state, st)) != cudaSuccess) return e;
    if ((e = launch_sort_pass<5>(key, idx, 1, n, nblk, dbase, ticket, state, st)) != cudaSuccess) return e;
    if ((e = launch_sort_pass<6>(key, idx, 0, n, nblk, dbase, ticket, state, st)) != cudaSuccess) return e;
    return launch_sort_pass<7>(key, idx, 1, n, nblk, dbase, ticket, state, st);
}

// ------------------------------------------------------------------------------------------
// S3 gather into key order as float4 (x,y,z,m): the "structure" the interaction kernels stage.
// Source: the float4 copy keygen wrote in the caller's order (one aligned 16-byte read per body).
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) gather_kernel(const float4* __restrict__ bin, const uint32_t* __restrict__ perm, int64_t n,
                                                     float4* __restrict__ body) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    body[i] = __ldg(bin + perm[i]);
}
cudaError_t launch_gather(const float4* bin, const uint32_t* perm, int64_t n, float4* body, cudaStream_t st) {
    HOT_LAUNCHED(1);
    gather_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(bin, perm, n, body);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// S4/S5 tree from the sorted keys in one sweep.
// For sorted position i:
//   b_i      = level at which key[i-1] and key[i] first differ (0 for i = 0, 22 if equal)
//   Lleaf_i  = level of the leaf holding i   = min(21, 1 + max_{j in [i-NLEAF,i]} cpl(key[j], key[j+NLEAF]))
//   Lgroup_i = level of the sink group of i  = same with NCRIT
// (cpl = number of common leading 3-bit digits; a level-L cell holds more than W bodies iff some
//  window of W+1 consecutive sorted keys containing i shares its first L digits.)
// A cell (l, i) -- level l, first body i -- exists iff b_i <= l <= Lleaf_i; in level-major order its
// index is level_base[l] + #{i' < i : b_i' <= l <= Lleaf_i'} (ascending numeric key order, C-4).
// ------------------------------------------------------------------------------------------
#define TREE_TILE 1024
#define TREE_ROWS (HOT_NLEVELS + 2) // 22 level rows, row 22 = groups, row 23 = leaves
int64_t tree_num_blocks(int64_t n) { return (n + TREE_TILE - 1) / TREE_TILE; }

__device__ __forceinline__ int first_diff_level(uint64_t a, uint64_t b) { // 1..21, 22 if equal
    uint64_t x = a ^ b;
    if (x == 0) return 22;
    int p = 63 - __clzll((long long)x);
    return 21 - p / 3;
}

// 32 x 32 bit matrix across the warp: lane r gives row r, lane c receives column c (bit r = bit c of row r)
__device__ __forceinline__ uint32_t transpose32(uint32_t x, int lane) {
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) {
        const uint32_t m = s == 16 ? 0x0000ffffu : s == 8 ? 0x00ff00ffu : s == 4 ? 0x0f0f0f0fu : s == 2 ? 0x33333333u : 0x55555555u;
        const uint32_t y = __shfl_xor_sync(FULL, x, s);
        x = (lane & s) ? ((x & ~m) | ((y >> s) & m)) : ((x & m) | ((y << s) & ~m));
    }
    return x;
}

__global__ void __launch_bounds__(TREE_TILE) tree_levels_kernel(const uint64_t* __restrict__ skey, int64_t n, int nleaf, int ncrit,
                                                                uint32_t* __restrict__ plev, uint32_t* __restrict__ counts, int64_t nblk) {
    __shared__ uint64_t sk[TREE_TILE + 2 * HOT_MAX_NCRIT];
    // v_q = 1 + cpl(key[q'], key[q'+W]) (0 outside the array), q' = T0 - W + q: plain (W < 32), or its prefix maximum inside
    // 32-element chunks (sp) with the chunk maxima (sc); the suffix maximum of a thread's own element stays in a register
    __shared__ uint8_t sp[TREE_TILE + HOT_MAX_NCRIT + 32], sc[(TREE_TILE + HOT_MAX_NCRIT) / 32 + 2];
    __shared__ uint32_t cnt[TREE_ROWS];
    const int tid = threadIdx.x, lane = tid & 31;
    const int64_t T0 = (int64_t)blockIdx.x * TREE_TILE;
    const int H = ncrit; // halo on both sides
    for (int p = tid; p < TREE_TILE + 2 * H; p += TREE_TILE) {
        int64_t g = T0 - H + p;
        sk[p] = (g >= 0 && g < n) ? skey[g] : 0ull;
    }
    if (tid < TREE_ROWS) cnt[tid] = 0;
    __syncthreads();
    const int64_t i = T0 + tid;
    const bool valid = i < n;
    int lev[2];
#pragma unroll
    for (int which = 0; which < 2; ++which) {
        const int W = which ? ncrit : nleaf;
        const int L = TREE_TILE + W;
        // the level of body i is the maximum of v over q in [tid, tid + W]
        int v[2];
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            const int q = tid + r * TREE_TILE;
            const int64_t g = T0 - W + q;
            v[r] = (q < L && g >= 0 && g + W < n) ? first_diff_level(sk[q + H - W], sk[q + H]) : 0;
        }
        int D;
        if (W < 32) { // short window: read it
            sp[tid] = (uint8_t)v[0];
            if (tid < W) sp[tid + TREE_TILE] = (uint8_t)v[1];
            __syncthreads();
            D = v[0];
            for (int j = 1; j <= W; ++j) D = max(D, (int)sp[tid + j]);
        } else { // long window: rest of the own chunk, whole chunks, start of the last chunk
            int suf = v[0];
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                if (r == 1 && (tid & ~31) >= W) break; // warp-uniform: no element of this warp lies below L
                int s = v[r], p = v[r];
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) { // out-of-range lanes return the caller's own value
                    s = max(s, __shfl_down_sync(FULL, s, o));
                    p = max(p, __shfl_up_sync(FULL, p, o));
                }
                const int q = tid + r * TREE_TILE;
                sp[q] = (uint8_t)p;
                if (lane == 0) sc[q >> 5] = (uint8_t)s;
                if (r == 0) suf = s;
            }
            __syncthreads();
            const int qe = tid + W;
            D = max(suf, (int)sp[qe]);
            for (int c = (tid >> 5) + 1; c < (qe >> 5); ++c) D = max(D, (int)sc[c]);
        }
        lev[which] = min(HOT_MAXLEVEL, D);
        __syncthreads();
    }
    int b = 0;
    if (valid && i > 0) b = first_diff_level(sk[tid + H - 1], sk[tid + H]);
    const int Lleaf = lev[0], Lgroup = lev[1];
    if (valid) plev[i] = (uint32_t)b | ((uint32_t)Lleaf << 8) | ((uint32_t)Lgroup << 16);
    // cells (l, i), b <= l <= Lleaf, counted per level: the lanes' level masks transposed give one level per lane
    const uint32_t col = transpose32((valid && b <= Lleaf) ? (2u << Lleaf) - (1u << b) : 0u, lane);
    if (lane < HOT_NLEVELS && col) atomicAdd(&cnt[lane], (uint32_t)__popc(col));
    {
        uint32_t m = __ballot_sync(FULL, valid && b <= Lgroup);
        if (lane == 0 && m) atomicAdd(&cnt[HOT_NLEVELS], (uint32_t)__popc(m));
        m = __ballot_sync(FULL, valid && b <= Lleaf);
        if (lane == 0 && m) atomicAdd(&cnt[HOT_NLEVELS + 1], (uint32_t)__popc(m));
    }
    __syncthreads();
    if (tid < TREE_ROWS) counts[(int64_t)tid * nblk + blockIdx.x] = cnt[tid];
}
cudaError_t launch_tree_levels(const uint64_t* skey, int64_t n, int nleaf, int ncrit, uint32_t* plev, uint32_t* counts, cudaStream_t st) {
    int64_t nblk = tree_num_blocks(n);
    HOT_LAUNCHED(1);
    tree_levels_kernel<<<(unsigned)nblk, TREE_TILE, 0, st>>>(skey, n, nleaf, ncrit, plev, counts, nblk);
    return cudaGetLastError();
}
cudaError_t launch_tree_scan(uint32_t* counts, int64_t nblk, uint32_t* totals, cudaStream_t st) {
    HOT_LAUNCHED(1);
    scan_rows_kernel<<<TREE_ROWS, 1024, 0, st>>>(counts, nblk, totals);
    return cudaGetLastError();
}

__device__ __forceinline__ uint64_t hash64(uint64_t k) {
    k ^= k >> 33; k *= 0xff51afd7ed558ccdull; k ^= k >> 33; k *= 0xc4ceb9fe1a85ec53ull; k ^= k >> 33;
    return k;
}
__device__ __forceinline__ uint64_t hash_slot(uint64_t key, uint64_t hmask) { return hash64(key) & hmask; } // home slot of a cell key
struct LevelBase { int64_t v[HOT_NLEVELS + 1]; };

__global__ void __launch_bounds__(TREE_TILE) tree_emit_kernel(const uint64_t* __restrict__ skey, const uint32_t* __restrict__ plev,
                                                              const uint32_t* __restrict__ counts, int64_t n, int64_t nblk, LevelBase LB,
                                                              uint64_t* __restrict__ ckey, uint32_t* __restrict__ cfirst,
                                                              uint32_t* __restrict__ ccount, int32_t* __restrict__ cchild,
                                                              int32_t* __restrict__ cparent,
                                                              GroupRec* __restrict__ group, int32_t* __restrict__ leafcell,
                                                              int2* __restrict__ open) {
    // per level (row 22: groups, row 23: leaves) and warp, as lane masks: which bodies start a cell of the level; which
    // bodies differ from their predecessor at or above the level (= where the cells of the level can end)
    __shared__ uint32_t sE[HOT_NLEVELS + 2][32], sB[HOT_NLEVELS][32];
    __shared__ uint32_t wpre[HOT_NLEVELS + 2][32]; // cells of the level in the earlier warps of the tile
    __shared__ uint32_t boff[HOT_NLEVELS + 2];     // ... and in the earlier tiles
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int64_t T0 = (int64_t)blockIdx.x * TREE_TILE;
    const int64_t i = T0 + tid;
    const bool valid = i < n;
    const uint32_t pl = valid ? plev[i] : 0u; // past the end: "differs at level 0", so that every cell ends at n
    const int b = (int)(pl & 255u), Lleaf = valid ? (int)((pl >> 8) & 255u) : -1, Lgroup = valid ? (int)((pl >> 16) & 255u) : -1;
    const bool starts = valid && b <= Lleaf;
    const uint32_t lt = (1u << lane) - 1u;
    {
        const uint32_t colE = transpose32(starts ? (2u << Lleaf) - (1u << b) : 0u, lane);
        const uint32_t colB = transpose32(~((1u << b) - 1u), lane);
        if (lane < HOT_NLEVELS) { sE[lane][w] = colE; sB[lane][w] = colB; }
        const uint32_t gm = __ballot_sync(FULL, valid && b <= Lgroup);
        const uint32_t lm = __ballot_sync(FULL, starts); // a leaf starts wherever a cell starts: the cell (Lleaf, i)
        if (lane == 0) { sE[HOT_NLEVELS][w] = gm; sE[HOT_NLEVELS + 1][w] = lm; }
    }
    if (tid <= HOT_NLEVELS + 1) boff[tid] = counts[(int64_t)tid * nblk + blockIdx.x];
    if (tid < HOT_NLEVELS) open[(int64_t)blockIdx.x * HOT_NLEVELS + tid] = make_int2(-1, -1);
    __syncthreads();
    if (w <= HOT_NLEVELS + 1) { // warp l: exclusive prefix of row l over the warps
        const uint32_t c = (uint32_t)__popc(sE[w][lane]);
        uint32_t x = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(FULL, x, o); if (lane >= o) x += y; }
        wpre[w][lane] = x - c;
    }
    __syncthreads();
    uint32_t gcount = 0; int32_t gcell = -1;
    const int64_t grank = (int64_t)boff[HOT_NLEVELS] + wpre[HOT_NLEVELS][w] + __popc(sE[HOT_NLEVELS][w] & lt); // if a group starts here
    if (starts) {
        const uint64_t mykey = skey[i];
        int32_t prev_cell = -1; // cell (l-1, i)
#pragma unroll 1
        for (int l = b; l <= Lleaf; ++l) {
            const int32_t c = (int32_t)(LB.v[l] + boff[l] + wpre[l][w] + __popc(sE[l][w] & lt));
            const int sh = 63 - 3 * l;
            const uint64_t ck = mykey >> sh;
            // end of the cell: the next body that differs from its predecessor at level <= l, found in the tile's masks;
            // the one cell per level that runs past the tile is left to tree_open_kernel (count 0 for now)
            int64_t hi;
            if (l == 0) hi = n;
            else {
                uint32_t m = sB[l][w] & ~(lt | (1u << lane));
                int ww = w;
                while (m == 0u && ++ww < 32) m = sB[l][ww];
                if (m) hi = T0 + (ww << 5) + __ffs((int)m) - 1;
                else { hi = i; open[(int64_t)blockIdx.x * HOT_NLEVELS + l] = make_int2(c, l == Lgroup ? (int)grank : -1); }
            }
            const uint32_t cnt = (uint32_t)(hi - i);
            ckey[c] = ck; cfirst[c] = (uint32_t)i; ccount[c] = cnt;
            int32_t parent = -1;
            if (l > b) parent = prev_cell;
            else if (l > 0) parent = (int32_t)(LB.v[l - 1] + boff[l - 1] + wpre[l - 1][w] + __popc(sE[l - 1][w] & (lt | (1u << lane)))) - 1;
            cparent[c] = parent;
            if (l == Lleaf) { cchild[c] = -1; leafcell[(int64_t)boff[HOT_NLEVELS + 1] + wpre[HOT_NLEVELS + 1][w] + __popc(sE[HOT_NLEVELS + 1][w] & lt)] = c; }
            if (prev_cell >= 0) cchild[prev_cell] = c; // cell (l-1, i) is internal: its first child starts at i too
            prev_cell = c;
            if (l == Lgroup) { gcount = cnt; gcell = c; }
        }
    }
    if (valid && b <= Lgroup) {
        GroupRec g; g.first = (uint32_t)i; g.count = gcount; g.cell = (uint32_t)gcell; g.pad = 0;
        group[grank] = g;
    }
}
// the cells that run past the tile of their first body (at most one per level and tile): end by gallop + bisection
// over the sorted keys, one cell per thread
__global__ void __launch_bounds__(256) tree_open_kernel(const int2* __restrict__ open, int64_t nslots, const uint64_t* __restrict__ skey, int64_t n,
                                                        const uint32_t* __restrict__ cfirst, uint32_t* __restrict__ ccount,
                                                        GroupRec* __restrict__ group) {
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nslots) return;
    const int2 e = open[s];
    if (e.x < 0) return;
    const int l = (int)(s % HOT_NLEVELS);
    const int sh = 63 - 3 * l;
    const int64_t i = cfirst[e.x];
    const uint64_t ck = skey[i] >> sh;
    const int64_t from = (s / HOT_NLEVELS) * TREE_TILE + TREE_TILE - 1; // the tile's last body is inside the cell
    int64_t lo = from, step = 1, p = from + 1;
    while (p < n && (skey[p] >> sh) == ck) { lo = p; step <<= 1; p = from + step; }
    int64_t hi = p < n ? p : n;
    while (hi - lo > 1) {
        int64_t mid = (lo + hi) >> 1;
        if ((skey[mid] >> sh) == ck) lo = mid; else hi = mid;
    }
    ccount[e.x] = (uint32_t)(hi - i);
    if (e.y >= 0) group[e.y].count = (uint32_t)(hi - i);
}
cudaError_t launch_tree_emit(const TreeEmitArgs& a, cudaStream_t st) {
    LevelBase LB;
    for (int l = 0; l <= HOT_NLEVELS; ++l) LB.v[l] = a.level_base[l];
    HOT_LAUNCHED(2);
    tree_emit_kernel<<<(unsigned)a.nblk, TREE_TILE, 0, st>>>(a.skey, a.plev, a.counts, a.n, a.nblk, LB, a.ckey, a.cfirst, a.ccount,
                                                             a.cchild, a.cparent, a.group, a.leafcell, a.open);
    const int64_t nslots = a.nblk * HOT_NLEVELS;
    tree_open_kernel<<<(unsigned)((nslots + 255) / 256), 256, 0, st>>>(a.open, nslots, a.skey, a.n, a.cfirst, a.ccount, a.group);
    return cudaGetLastError();
}
// The hash table key -> cell, open addressing with linear probing.  A slot holds the cell INDEX only
// (-1 = free): the key it stands for is ckey[index], which a lookup compares against -- so an insert is one 32-bit CAS
// and the table is 4 bytes per slot (33-67 MB at 2^24 bodies: L2-resident; with keys stored beside the indices it was
// 201 MB and every insert two DRAM sector read-modify-writes).  One independent insert per thread.
__global__ void __launch_bounds__(256) tree_link_kernel(const uint64_t* __restrict__ ckey, int64_t ncells, int32_t* __restrict__ hval,
                                                        int64_t hmask, int* __restrict__ maxprobe) {
    __shared__ int s_probe;
    if (threadIdx.x == 0) s_probe = 0;
    __syncthreads();
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int probe = 0;
    if (c < ncells) {
        uint64_t h = hash_slot(ckey[c], (uint64_t)hmask);
        while (atomicCAS(&hval[h], -1, (int32_t)c) != -1) { h = (h + 1) & (uint64_t)hmask; ++probe; }
    }
    // longest probe sequence: one global atomic per block at most (every thread reading the one counter queues in its L2 slice)
    probe = __reduce_max_sync(FULL, probe);
    if ((threadIdx.x & 31) == 0 && probe > 0) atomicMax(&s_probe, probe);
    __syncthreads();
    if (threadIdx.x == 0 && s_probe > 0 && s_probe > *((volatile int*)maxprobe)) atomicMax(maxprobe, s_probe);
}
cudaError_t launch_tree_link(const uint64_t* ckey, int64_t ncells, int32_t* hval, int64_t hmask, int* maxprobe, cudaStream_t st) {
    HOT_LAUNCHED(1);
    tree_link_kernel<<<(unsigned)((ncells + 255) / 256), 256, 0, st>>>(ckey, ncells, hval, hmask, maxprobe);
    return cudaGetLastError();
}
// per cell: the child mask (the children are the cells from cchild on whose key is this key extended by one octant:
// at most eight consecutive, sorted keys -- no atomics) and the 16-byte record the walk reads
__global__ void __launch_bounds__(256) tree_finalize_kernel(const uint64_t* __restrict__ ckey, const uint32_t* __restrict__ cfirst,
                                                            const uint32_t* __restrict__ ccount, uint32_t* __restrict__ cmask,
                                                            const int32_t* __restrict__ cchild, WalkCell* __restrict__ wc,
                                                            int64_t ncells, int* __restrict__ errflag) {
    int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncells) return;
    uint64_t k = ckey[c];
    int level = (63 - __clzll((long long)k)) / 3;
    uint64_t mort = k & ((1ull << (3 * level)) - 1ull);
    int up = HOT_MAXLEVEL - level;
    uint64_t ox = (uint64_t)compact21(mort >> 2) << up, oy = (uint64_t)compact21(mort >> 1) << up, oz = (uint64_t)compact21(mort) << up;
    const int32_t ch = cchild[c];
    bool leaf = ch < 0;
    uint32_t mask = 0;
    if (!leaf) {
#pragma unroll 1
        for (int j = 0; j < 8 && ch + j < ncells; ++j) {
            const uint64_t kk = ckey[ch + j];
            if ((kk >> 3) != k) break;
            mask |= 1u << (uint32_t)(kk & 7ull);
        }
    }
    cmask[c] = mask;
    uint32_t cnt = leaf ? ccount[c] : (uint32_t)__popc(mask);
    if (cnt >= (1u << 27)) { atomicOr(errflag, 2); cnt = (1u << 27) - 1; }
    uint64_t packed = ox | (oy << 21) | (oz << 42) | (leaf ? (1ull << 63) : 0ull);
    WalkCell r;
    r.x = (uint32_t)packed; r.y = (uint32_t)(packed >> 32);
    r.z = leaf ? cfirst[c] : (uint32_t)ch;
    r.w = ((uint32_t)level << 27) | cnt;
    wc[c] = r;
}
cudaError_t launch_tree_finalize(const uint64_t* ckey, const uint32_t* cfirst, const uint32_t* ccount, uint32_t* cmask,
                                 const int32_t* cchild, WalkCell* wc, int64_t ncells, int* errflag, cudaStream_t st) {
    HOT_LAUNCHED(1);
    tree_finalize_kernel<<<(unsigned)((ncells + 255) / 256), 256, 0, st>>>(ckey, cfirst, ccount, cmask, cchild, wc, ncells, errflag);
    return cudaGetLastError();
}
__global__ void hash_lookup_kernel(const uint64_t* __restrict__ ckey, const int32_t* __restrict__ hval, int64_t hmask,
                                   const uint64_t* __restrict__ keys, int64_t nkeys, int32_t* __restrict__ out) {
    int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= nkeys) return;
    uint64_t k = keys[q];
    int32_t r = -1;
    if (k != 0) {
        uint64_t h = hash_slot(k, (uint64_t)hmask);
        while (true) {
            const int32_t v = hval[h];
            if (v < 0) break;
            if (ckey[v] == k) { r = v; break; }
            h = (h + 1) & (uint64_t)hmask;
        }
    }
    out[q] = r;
}
cudaError_t launch_hash_lookup(const uint64_t* ckey, const int32_t* hval, int64_t hmask, const uint64_t* keys, int64_t nkeys,
                               int32_t* out, cudaStream_t st) {
    if (nkeys > 0) hash_lookup_kernel<<<(unsigned)((nkeys + 255) / 256), 256, 0, st>>>(ckey, hval, hmask, keys, nkeys, out);
    return cudaGetLastError();
}

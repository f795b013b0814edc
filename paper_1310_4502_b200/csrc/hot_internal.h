// Internal declarations shared by the translation units of libhot (CUDA, sm_100a).
// Not part of the public boundary (include/hot.h) and never seen by the oracle.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "hot.h"

extern long long g_hot_launches; // kernels launched by the library since the last reset (hot_stats)
#define HOT_LAUNCHED(k) (g_hot_launches += (k))

#define HOT_MAXLEVEL 21
#define HOT_NLEVELS 22        // levels 0..21
#define HOT_MAX_NCRIT 256
#define HOT_MAX_NLEAF 32

// 16-byte record the walk reads per visited cell (S7).
//   x: ox | oy<<21 (low 11 bits of oy)          packed 63-bit integer corner on the 2^21 grid
//   y: oy>>11 | oz<<10 | leaf<<31
//   z: first child (internal) or first body (leaf)
//   w: level<<27 | count  (count = number of children, or of bodies for a leaf; < 2^27)
struct __align__(16) WalkCell { uint32_t x, y, z, w; };

// per-cell expansion data (S6), gathered when a cell is accepted
struct __align__(16) CellA { double zx, zy, zz; float m0; float bmax; }; // centre of mass, mass, b_max: radius about the centre of mass that holds every body (R-15)
struct __align__(16) CellM2 { float xx, xy, xz, yy, yz, zz, t2, pad1; };     // t2 = trace
// the same record as the P-C kernel stages it (cellE2): 3 xx, 3 xy, 3 xz, 3 yy, 3 yz, 3 zz, 1.5 t2, 0.5 t2 -- the
// constant factors of the order-2 terms folded in once per cell instead of once per interaction
// order 4: M3 (10) + M4 (15) + traces t3 (3), T4 (6), t4 (1) = 35 floats -> 36
struct __align__(16) CellM34 { float v[36]; };

struct GroupRec { uint32_t first, count, cell, pad; };

struct Tree {
    int64_t n = 0;
    int periodic = 0, nleaf = 16, ncrit = 256;
    hot_box box{};
    double lo[3], size;
    // bodies
    uint64_t* key[2] = {nullptr, nullptr};   // ping-pong, key[0] holds the sorted keys after build
    uint32_t* idx[2] = {nullptr, nullptr};   // idx[0] = perm
    float4* body = nullptr;                  // key-ordered (x,y,z,m)
    float4* bin = nullptr;                   // the same records in the caller's order (written by keygen, read by the gather)
    uint32_t* plev = nullptr;                // per body: b | Lleaf<<8 | Lgroup<<16
    // cells
    int64_t ncells = 0, nleaves = 0, ngroups = 0;
    int max_level = 0;
    int64_t level_base[HOT_NLEVELS + 1];
    uint64_t* ckey = nullptr;
    uint32_t *cfirst = nullptr, *ccount = nullptr, *cmask = nullptr;
    int32_t *cchild = nullptr, *cparent = nullptr;
    int32_t* leafcell = nullptr;             // [nleaves] cell index of every leaf, in body order (the upward pass starts here)
    WalkCell* wcell = nullptr;
    GroupRec* group = nullptr;
    uint32_t *glpc = nullptr, *glpp = nullptr, *glvis = nullptr; // per group, last walk: accepted cells, listed bodies (without the group's own), cells visited
    unsigned long long *pcoff = nullptr, *ppoff = nullptr; // [ngroups] start of each group's lists in the arena
    // hash
    int64_t hcap = 0;
    int32_t* hval = nullptr;                 // slot -> cell index or -1; the slot's key is ckey[index]
    int hash_max_probe = 0;
    // periodic far field: polynomial of the sink position (hot_periodic.cu)
    bool far_ready = false;
    double farD[165];
    double* far = nullptr;                   // [n][4] far field per body, key order
    double* farc = nullptr;                  // [n][4] far field + fp64 coarse-cell monopoles of the current hot_forces call
    // moments
    int mom_order = -1;
    CellA* cellA = nullptr;
    CellM2* cellM2 = nullptr;
    CellM2* cellE2 = nullptr; // evaluation form of cellM2 (see CellM2)
    CellM34* cellM34 = nullptr;
    float *cellHiRaw = nullptr, *cellHiT = nullptr; // orders 6, 8 (f-3): raw moments of degree 5.. and their trace record, per cell, in units of the cell side
    int hi_order = 0;                        // order those two were built for (their per-cell strides follow from it)
    // f-1 (background subtraction, periodic): per cell, moments about the cell centre minus the uniform cube's
    double* cellM0d = nullptr;               // periodic: cell masses in fp64 (upward pass)
    float4* bgA = nullptr; CellM2* bgE2 = nullptr; CellM34* bgM34 = nullptr; int bg_order = -1;
    double total_mass = 0.0;                 // sum of the masses in fp64 (the far field's zeroth moment)
    uint32_t* glpv = nullptr; unsigned long long* gpvoff = nullptr; // per group: accepted virtual cubes, where they start
    float4* cellMac = nullptr;               // order 4 only: b, 3 B2, 4 sqrt(B2 B4), 6 b B4 (the error bounds of R-16, numerators)
    uint32_t *glpc0 = nullptr, *glpc2 = nullptr; // per group, tolerance mode: accepted monopoles, quadrupoles
};

// ---- build stages (hot_build.cu) ------------------------------------------------------------
// every launcher returns the cudaError_t of its last launch; all work goes to `st`
cudaError_t launch_keygen(const float* pos, const float* mass, int64_t n, float lox, float loy, float loz, float inv,
                          uint64_t* key, float4* bin, uint32_t* hist, int* errflag, cudaStream_t st);
// launch_keygen also clears the sort's scratch `hist` and counts the eight digit histograms of the keys into it.
// sorts (key, position) pairs stably, ascending: idx[0] need not be initialised (the first pass takes a key's index from
// its position); result ends in key[0]/idx[0]; scratch: hist of sort_hist_elems(n) u32
size_t sort_hist_elems(int64_t n);
cudaError_t launch_radix_sort(uint64_t* key[2], uint32_t* idx[2], int64_t n, uint32_t* hist, cudaStream_t st);
cudaError_t launch_gather(const float4* bin, const uint32_t* perm, int64_t n, float4* body, cudaStream_t st);
// tree pass 1: per-body levels + per-block per-level counts.  counts: [HOT_NLEVELS+1][nblk] u32
int64_t tree_num_blocks(int64_t n);
cudaError_t launch_tree_levels(const uint64_t* skey, int64_t n, int nleaf, int ncrit, uint32_t* plev,
                               uint32_t* counts, cudaStream_t st);
// exclusive scan of each row of counts over blocks; totals[row]
cudaError_t launch_tree_scan(uint32_t* counts, int64_t nblk, uint32_t* totals, cudaStream_t st);
struct TreeEmitArgs {
    const uint64_t* skey; const uint32_t* plev; const uint32_t* counts; int64_t n, nblk;
    int64_t level_base[HOT_NLEVELS + 1];
    uint64_t* ckey; uint32_t* cfirst; uint32_t* ccount; int32_t* cchild; int32_t* cparent;
    GroupRec* group; int32_t* leafcell;
    int2* open; // [nblk][HOT_NLEVELS] scratch: the cells whose end lies beyond the tile of their first body
};
cudaError_t launch_tree_emit(const TreeEmitArgs& a, cudaStream_t st);
cudaError_t launch_tree_link(const uint64_t* ckey, int64_t ncells, int32_t* hval, int64_t hmask, int* maxprobe, cudaStream_t st);
cudaError_t launch_tree_finalize(const uint64_t* ckey, const uint32_t* cfirst, const uint32_t* ccount,
                                 uint32_t* cmask /* out */, const int32_t* cchild, WalkCell* wc,
                                 int64_t ncells, int* errflag, cudaStream_t st);
cudaError_t launch_hash_lookup(const uint64_t* ckey, const int32_t* hval, int64_t hmask,
                               const uint64_t* keys, int64_t nkeys, int32_t* out, cudaStream_t st);

// ---- upward pass (hot_moments.cu) -------------------------------------------------------------
cudaError_t launch_moments(const Tree& t, int order, cudaStream_t st);

// ---- walk (hot_walk.cu): emits the interaction lists of the groups [g0, g1) ---------------------------
// While a group is walked its particle-particle list is kept as RUNS of bodies, first | (count-1) << 27
// with count <= 32 (one per rejected leaf; a finest-level leaf with more bodies gives several); the
// runs are expanded to one body index per entry when the list moves to the arena.
#define HOT_RUN_SHIFT 27
// Periodic boxes: accepted cells of levels <= HOT_COARSE_LEVEL carry HOT_COARSE_FLAG in the cell list.  They are
// few (~1250 per group at theta = 0.5) but hold the large, nearly cancelling part of the image sum, so their
// monopole terms are evaluated in fp64 by coarse_monopole_kernel and left out of the fp32 kernel (R-14).
#define HOT_COARSE_LEVEL 3
#define HOT_COARSE_FLAG 0x80000000u
struct WalkArgs {
    const WalkCell* wcell; const GroupRec* group; int64_t g0, g1;
    unsigned long long mac_t[HOT_NLEVELS]; // accept a level-l cell iff d2 >= mac_t[l] (R-7, "MAC table")
    int periodic;
    uint32_t *lpc, *lpp, *lvis;            // per group: accepted cells, bodies of rejected leaves, cells visited
    unsigned long long *pcoff, *ppoff;     // per group: where its two lists start in the arena
    uint32_t* pclist; uint32_t* pplist;    // the arena: cell indices / body indices
    uint8_t* pcimg; uint8_t* ppimg;        // periodic: image id (0..124) of every list entry
    unsigned long long cappc, cappp;       // arena capacity in entries
    unsigned long long* tops;              // [0], [1]: entries handed out so far
    int* first_fail;                       // smallest group that did not fit the arena (INT_MAX: none)
    uint32_t* stage; uint8_t* stage_img; int64_t stage_cap; // per-warp staging: [2][stage_cap] entries
    unsigned int* counter;                 // dynamic group scheduler
    unsigned long long* stat;              // [1] ring spills
    uint32_t* gstack; int64_t gstack_cap;  // per-warp spill arena (entries per warp)
    int* errflag;                          // bit 2: spill arena exhausted, bit 3: staging too small
    // error-bound criterion (tolmode != 0; R-16): accept at the cheapest order whose bound is <= tol
    int tolmode; double tol; double lo[3], size;
    double hreal;                          // spline softening: h (an accepted cell lies wholly beyond it), else 0
    const CellA* cellA; const float4* cellMac;   // per cell: centre of mass / (b, 3 B2, 4 sqrt(B2 B4), 6 b B4)
    uint32_t *lpc0, *lpc2;                 // per group: accepted monopoles, quadrupoles (the list is ordered mono | quad | hexa)
    // background subtraction (bgmode != 0, periodic; R-18): lpc0 / lpc2 = plain / background-subtracted cells
    int bgmode; const uint32_t* cmask;
    uint4* vstack; int64_t vstack_cap;     // per warp: virtual cubes still to look at
    uint4* vstage; int64_t vstage_cap;     // per warp: accepted virtual cubes of the group being walked
    uint4* pvlist; unsigned long long cappv; // arena of the accepted virtual cubes (tops[2]); per group lpv, pvoff
    uint32_t* lpv; unsigned long long* pvoff;
};
int walk_grid_warps();
cudaError_t launch_walk(const WalkArgs& a, cudaStream_t st);
// stat[0] += cells visited, stat[2] += sum n_G (L_pp + n_G), stat[3] += sum n_G L_pc over the groups [0, ng);
// with lpc0 / lpc2 (tolerance mode): stat[4], stat[5] += sum n_G x accepted monopoles / quadrupoles
cudaError_t launch_group_stats(const GroupRec* group, const uint32_t* lpc, const uint32_t* lpp, const uint32_t* lvis,
                               const uint32_t* lpc0, const uint32_t* lpc2, int64_t ng, unsigned long long* stat, cudaStream_t st);

// ---- interactions (hot_forces.cu): evaluates the lists of the groups [g0, g1) -------------------------
struct ForceArgs {
    const WalkCell* wcell; const CellA* cellA; const CellM2* cellE2; const CellM34* cellM34;
    const float4* body; const uint32_t* perm; const GroupRec* group; int64_t g0, g1;
    const unsigned long long* pcoff; const unsigned long long* ppoff; const uint32_t* lpc; const uint32_t* lpp;
    const uint32_t* pclist; const uint32_t* pplist; const uint8_t* pcimg; const uint8_t* ppimg;
    const double* far;            // periodic: far field (ax, ay, az, phi) per body in key order, added in fp64; else NULL
    float eps2; int order; int periodic;
    int spline; float hinv;       // f-4: cubic-spline softening with h = 2.8 eps instead of Plummer; 1 / h
    double lo[3], size;
    float* acc; float* pot;
    unsigned int* counter;        // dynamic scheduler over the work items
    uint4* items;                 // one per pass of a group, ordered by sinks per lane (launch_plan)
    unsigned int* cls;            // plan_cls_elems(g1 - g0, sb_shift) words: per-(superblock, class) counts, starts, cursors, total
    // tolerance mode: one launch per order over its segment of the cell lists (seg = 0, 1, 2; -1: the whole list)
    int seg; const uint32_t *lpc0, *lpc2; int do_pp, accumulate;
    // background subtraction: bgv = 1 evaluates the flagged cells (seg 1) from these records into out_farc[body][4] (fp64)
    int bgv; const float4* bgA; const CellM2* bgE2; const CellM34* bgM34; double* out_farc;
    int sb_shift; unsigned int nsb; // 2^sb_shift groups per superblock (>= 8), number of superblocks of [g0, g1)
};
size_t plan_cls_elems(int64_t ngroups, int sb_shift);
cudaError_t launch_plan(const ForceArgs& a, cudaStream_t st);   // fills items / cls for groups [g0, g1)
cudaError_t launch_forces(const ForceArgs& a, cudaStream_t st); // after launch_plan

// ---- periodic far field (hot_periodic.cu) ------------------------------------------------------------
void far_coefficients(double* out165);                    // host: Taylor coefficients of psi_sm, degree-major
void far_sink_polynomial(const double* S, double* D);     // host: per-sink polynomial from the global moments
cudaError_t launch_far_moments(const Tree& t, double* S /*device [165]*/, cudaStream_t st);
cudaError_t launch_far_eval(const Tree& t, const double* D /*host [165]*/, double* far /*device [n][4], key order*/, cudaStream_t st);
// farc[body] = far[body] + fp64 monopole sum over the flagged cells of the body's group, groups [a.g0, a.g1)
cudaError_t launch_coarse_monopoles(const ForceArgs& a, const double* far, double* farc, double eps2, cudaStream_t st);

// ---- FP32 roofline denominator measured on the device (hot_peak.cu) ------------------------------------
// ---- f-1: per-cell background subtraction (hot_bg.cu) ---------------------------------------------------------
cudaError_t launch_bg_moments(const Tree& t, int order, double rhobar, cudaStream_t st);
// farc[body] = far[body] + background added back in closed form + flagged cells + virtual cubes, groups [a.g0, a.g1)
cudaError_t launch_forces_bg(const ForceArgs& a, const Tree& t, const double* far, double* farc, const uint4* pvlist, const uint32_t* lpv,
                             const unsigned long long* pvoff, double rhobar, int with_cells, cudaStream_t st);

// ---- f-3: the terms of degree 5 .. P (P = 6, 8) of every accepted cell, added to acc / pot (hot_hi.cu) ----------
int hi_record_floats(int order); int hi_raw_floats(int order);
cudaError_t launch_forces_hi(const ForceArgs& a, int P, const float* hiT, int hi_stride, cudaStream_t st);

// ---- f-4: kick and drift (hot_step.cu) -------------------------------------------------------------------
cudaError_t launch_kick_drift(float* pos, float* vel, const float* acc, int64_t n, float dtk, float dtd, float lox, float loy, float loz,
                              float size, int periodic, cudaStream_t st);

cudaError_t measure_fp32(double* tf_scalar, double* tf_packed, cudaStream_t st);
cudaError_t measure_fp32_operands(double* tf3, cudaStream_t st); // packed 2 register reads, packed 3, scalar 3

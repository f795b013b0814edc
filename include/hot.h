/*
 * hot.h -- C ABI of the B200-native hot path of 2HOT's hashed oct-tree method
 * (Warren, "2HOT: An Improved Parallel Hashed Oct-Tree N-Body Algorithm for Cosmological
 * Simulation", SC'13, arXiv:1310.4502; the text is PAPER.md, cited as PAPER.md:<line>).
 *
 * What the library computes (one GPU, every stage a CUDA kernel for sm_100a):
 *   hot_build : integer keys from coordinates ("mapping of spatial co-ordinates to
 *               integer keys described in WS93"), on-node radix sort, bodies into
 *               key order, the hashed oct-tree of the sorted keys and the sink
 *               cells of the m x n blocking.
 *   hot_forces: moments of eq (6), the source/sink traversal with a multipole
 *               acceptance criterion and the Plummer-softened
 *                particle-particle and Cartesian-multipole particle-cell
 *               interactions of eq (5) giving the right-hand side of eq (2)
 *               (PAPER.md:57): acc_i = -grad phi(x_i), phi_i, G = 1, self term excluded.
 *               Periodic boxes: 124 boundary cubes + local expansion, p = 8, ws = 2.
 *   hot_stats : sizes, interaction counts and per-stage device times of the last calls.
 *
 * The readings of everything the paper leaves open (key bit order, bucket sizes, the
 * opening criterion, the far-field route) are listed in DESIGN.md "Readings".
 *
 * Conventions
 *   - "device" pointers are CUDA device pointers of the current device (e.g. torch data_ptr());
 *     "host" pointers are ordinary host memory.  The library never keeps a caller pointer.
 *   - One implicit context per process.  Not thread-safe.
 *   - Every call returns HOT_OK (0) or a negative hot_status; hot_last_error() gives the text.
 *     No exceptions, no abort, no printing.  After a failed hot_build there is no build.
 *   - Work is enqueued on the stream given to hot_set_stream (default: the legacy stream 0).
 *     hot_build synchronises that stream (it needs the cell count to size the tree);
 *     hot_forces synchronises it once at the end to read the error flag.
 */
#ifndef HOT_H_
#define HOT_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    HOT_OK = 0,
    HOT_EINVAL = -1,  /* bad argument: NULL, n out of range, size <= 0, theta, eps, order */
    HOT_ERANGE = -2,  /* a particle lies outside [lo, lo+size)^3 (open AND periodic mode) */
    HOT_ENOMEM = -3,  /* device or host allocation failed */
    HOT_ECUDA = -4,   /* a CUDA call or kernel failed; text in hot_last_error() */
    HOT_EORDER = -5,  /* hot_forces / export before a successful hot_build */
    HOT_EINTERNAL = -6 /* traversal scratch exhausted or an internal invariant failed */
} hot_status;

/* Root cube of the tree and, when periodic, the period. size > 0. */
typedef struct {
    float lo[3];
    float size;
} hot_box;

/* Filled by hot_stats (host struct).  Times are device milliseconds of the LAST call that ran
 * the stage, measured with CUDA events on the library's stream. */
typedef struct {
    int64_t n, n_cells, n_leaves, n_groups;
    int32_t max_level, nleaf, ncrit, periodic;
    int64_t hash_capacity;
    int32_t hash_max_probe, order; /* order of the last hot_forces */
    /* sum over sink groups G of n_G * L_pp(G) and n_G * L_pc(G); L_pp counts the group's own
     * particles too (the self slot), images included when periodic */
    uint64_t pp_interactions, pc_interactions;
    uint64_t cells_visited;     /* MAC tests of the last walk */
    uint64_t walk_spills;       /* traversal-stack spills to the global arena */
    float ms_keygen, ms_sort, ms_gather, ms_tree, ms_moments;
    float ms_walk;   /* list walks: count pass + offset scan + fill pass(es) */
    float ms_eval;   /* particle-particle / particle-cell interaction kernels (the FP32-bound stage) */
    float ms_farfield;
    float ms_build_total, ms_forces_total;
    int32_t list_chunks; /* group chunks the lists were walked / evaluated in (1 unless the arena is short) */
    float ms_coarse;     /* periodic only: fp64 monopoles of the coarsest accepted cells (R-14) */
    uint64_t list_entries;      /* accepted cells + listed bodies over all groups (4 B each, +1 B when periodic) */
    int64_t bytes_allocated;
    int64_t launches_build, launches_forces; /* kernels launched by the last hot_build / hot_forces */
    /* pc_interactions by expansion order (sum over groups of n_G x accepted cells of that order): all in one entry after
     * hot_forces, a mix after hot_forces_tol ("hexadecapole ... quadrupole ... monopole interactions") */
    uint64_t pc_monopole, pc_quadrupole, pc_hexadecapole;
} hot_stats_t;

/* Bucket sizes of the tree: a cell with more than nleaf bodies is split (down
 * to level 21); sink groups are the cells with at most ncrit bodies whose parent has more.
 * 1 <= nleaf <= ncrit <= 256, nleaf <= 32.  Takes effect at the next hot_build.
 * Defaults: nleaf = 16, ncrit = 256 (measured fastest step on the N = 2^24 clustered set). */
int hot_set_params(int nleaf, int ncrit);

/* Upper bound in bytes on the interaction-list arena of hot_forces (0 = default: as much as fits in
 * ~70% of the free device memory).  When the lists of all sink groups do not fit, hot_forces walks and
 * evaluates the groups in chunks (hot_stats list_chunks); HOT_ENOMEM if one group alone does not fit. */
int hot_set_list_arena(int64_t max_bytes);

/* pos : device, [n][3] fp32 row-major x,y,z; borrowed.   mass: device, [n] fp32 > 0; borrowed.
 * n   : 1 <= n <= 2^27 (and < 2^27 coincident bodies in one finest-level cell).  The bound is the 27-bit count
 *       and 28-bit cell index of the 16-byte record the walk reads per cell; 2^27 fp32
 *       bodies with their lists are also what fits 180 GB.
 * periodic: 0 open, 1 periodic with period box.size.  In both modes every particle must satisfy
 *           0 <= fl32((x-lo)*fl32(1/size)) < 1 per axis, else HOT_ERANGE (the caller wraps).
 * Builds keys, the stable key-sorted permutation, key-ordered bodies, cells, hash table and
 * sink groups; replaces any previous build. */
int hot_build(const float* pos, const float* mass, int64_t n, hot_box box, int periodic);

/* theta: opening angle, 0 <= theta < 1 (0: every interaction is particle-particle).
 * eps  : Plummer softening length >= 0 (0 with coincident distinct bodies gives inf/NaN).
 * order: 0 (monopole), 2 (through quadrupole), 4 (through hexadecapole, octupole included), or 6 / 8: the terms of
 *        degree 5 .. order come from generated code (csrc/gen_hi_orders.py), an accuracy feature.
 * acc  : device, [n][3] fp32, caller's particle order; overwritten.
 * pot  : device, [n] fp32 or NULL; overwritten.
 * May be called repeatedly on one build with different theta / eps / order. */
int hot_forces(double theta, double eps, int order, float* acc, float* pot);

/* The same evaluation with the paper's kind of acceptance criterion: an ABSOLUTE bound on the acceleration error of each
 * accepted interaction, with the expansion order chosen per interaction ("MAC based on an absolute error",
 * 90-94 and Fig 3, 238: a mix of monopole, quadrupole and hexadecapole interactions).  The paper prints no formula; the
 * reading is DESIGN.md R-16: a cell of radius b_max about its centre of mass z with B_n = sum m |y - z|^n, at distance
 * R > b_max from the nearest point of the sink group's cube, truncated after order p, is off by at most
 * (p+2) B_(p+1) / (R^(p+1) (R - b_max)^2); the cheapest of monopole (p = 1 about the centre of mass), quadrupole and
 * hexadecapole whose bound is <= tol is taken, else the cell is opened (a leaf: its bodies interact directly).
 * tol: absolute acceleration error per interaction, in the caller's units (G = 1), >= 0 (0: only exact interactions).
 * The criterion compares floating-point numbers: list counts are reproducible run to run, but a borderline cell may
 * fall differently from another implementation of the same formulas.  Other arguments as hot_forces. */
int hot_forces_tol(double tol, double eps, float* acc, float* pot);

int hot_stats(hot_stats_t* out);

/* Softening kernel of the following hot_forces / hot_forces_tol calls ("Plummer or spline [50] kernel").
 * 0 (default): Plummer, g = (r^2 + eps^2)^(-1/2), also inside the expansions of accepted cells.
 * 1: the cubic-spline kernel of ref [50] with h = 2.8 eps (same central potential -m/eps): a body is a ball of radius
 *    h; pairs closer than h use the kernel's closed form, everything else is Newtonian.  An accepted cell must lie
 *    wholly beyond h from the sink group (integer geometry as in R-7; R-17), so the lists depend on eps.
 * (The compensating K1 kernel of ref [13], is not built: its formula is not in the paper.) */
int hot_set_softening(int kind);

/* Per-cell background subtraction for periodic boxes (Fig 2; R-18), 0 (default) or 1; applies to
 * the following hot_forces calls (orders 0, 2, 4; not hot_forces_tol).  Around each sink group a near cube (5 x 5 x 5
 * cells of the group's level) is walked as usual; a cell accepted outside it interacts through its moments about the
 * cell centre minus those of a cube of the mean density (same order, dipole included); empty octants and the cubes of
 * rejected leaves out there count as negative-background cubes; what was subtracted is added back in closed form (the
 * field of a homogeneous cube).  Same field as without it to the truncation error, without the cancellation of large
 * terms in fp32; L_pc of hot_export_groups then counts plain and background-subtracted cells together and
 * hot_export_group_orders returns (plain cells, background-subtracted cells, accepted negative-background cubes). */
int hot_set_background(int on);

/* The "kick" and "drift" operators of the leapfrog around the force call: vel += acc * dt_kick, then
 * pos += vel * dt_drift, one fp32 fused multiply-add each; periodic != 0 wraps pos into [lo, lo + size).  In a
 * comoving background the two factors are integrals over the expansion history: the caller's.
 * pos, vel: device, [n][3] fp32, updated in place; acc: device, [n][3]. */
int hot_kick_drift(float* pos, float* vel, const float* acc, int64_t n, float dt_kick, float dt_drift, hot_box box, int periodic);

/* Same path with HOST buffers: copies pos/mass to the device, hot_build, hot_forces, copies acc
 * (and pot unless NULL) back; returns after the results are in host memory. */
int hot_step_host(const float* pos, const float* mass, int64_t n, hot_box box, int periodic,
                  double theta, double eps, int order, float* acc, float* pot);

int hot_set_stream(void* cuda_stream); /* cudaStream_t; NULL = legacy default stream */
void hot_free(void);                   /* releases everything the library owns */
const char* hot_last_error(void);

/* Roofline denominator of the interaction kernels measured on the current device: TFLOP/s of a
 * register-only fused-multiply-add chain, scalar (FFMA) and packed pairs (FFMA2); FMA = 2 flops.
 * ~10 ms of device time on the library's stream.  Outputs: host. */
int hot_measure_fp32(double* tflops_scalar, double* tflops_packed);
/* The same pipe fed from the register file, which delivers 64 bits per lane and clock: TFLOP/s of fused multiply-adds
 * whose sources are [0] packed pairs, two different registers (a*a+d), [1] packed pairs, three different registers
 * (a*b+d), [2] scalar, three different registers.  [1] and [2] fall to 2/3 of the peak: the ceiling of the inner loops
 * of the interaction kernels, most of whose operands are per-sink registers.  tflops3: host, [3]. */
int hot_measure_fp32_operands(double* tflops3);

/* Host-only, needs no GPU: the 165 Taylor coefficients c_abc (a+b+c <= 8, degree-major, x exponent
 * descending then y; odd ones are zero) of psi_sm(r) = psi(r) - sum_{|n|_inf<=2} 1/|r-n| about r = 0, in
 * units of the box: the table of the periodic far field (p = 8, ws = 2).  coef165: host. */
int hot_far_coefficients(double* coef165);

/* ---- the ONE allocation-free entry point ------------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it): the
 * stable radix sort of hot_build (S2) on caller-provided buffers, its scratch (digit counts, tile tickets,
 * look-back state) in a fixed device array inside the library.  Calls no cudaMalloc / cudaFree / allocating routine.
 *   key      : device, [n] u64; in: the keys, out: sorted ascending
 *   perm     : device, [n] u32; out: perm[i] = input position of the i-th sorted key; equal keys keep ascending position
 *   key_work, idx_work : device, [n] u64 / u32 work buffers (contents undefined afterwards); none may alias another
 *   n        : 1 <= n <= 2^22 = 4,194,304 (the fixed scratch: 2.1 MB, held by every GPU that loads the library until
 *              exit); larger n: HOT_EINVAL with a message naming the limit (use hot_build)
 *   cuda_stream : cudaStream_t the work is enqueued on (NULL: legacy default stream); returns without synchronising
 * Every call shares the one scratch array (cleared at the start of each call, stream-ordered): calls that overlap on
 * the GPU -- two streams, two host threads -- race.  Error text: hot_noalloc_last_error(). */
int hot_sort_keys_noalloc(uint64_t* key, uint32_t* perm, uint64_t* key_work, uint32_t* idx_work, int64_t n, void* cuda_stream);
const char* hot_noalloc_last_error(void);

/* ---- introspection for the parity tests: HOST output arrays, caller-allocated -------------- */
/* sorted keys and the permutation: key_sorted[i] = key of caller's particle perm[i]; [n] each */
int hot_export_keys(uint64_t* key_sorted, uint32_t* perm);
/* cells in ascending numeric key order; any pointer may be NULL.  cap = array length;
 * *ncells is always set; HOT_EINVAL if cap is too small.
 * child = index of the first child or -1 for a leaf; parent = -1 for the root. */
int hot_export_cells(uint64_t* key, uint32_t* first, uint32_t* count, uint8_t* mask,
                     int32_t* child, int32_t* parent, int64_t cap, int64_t* ncells);
/* sink groups in particle order: index and key of the group's cell, its first body (sorted
 * position) and body count, and the list counts of the last hot_forces (zeros before the first):
 * L_pc = accepted cells, L_pp = particles of rejected leaves (the group's own bodies included), both
 * summed over the 125 images when periodic.  Any pointer may be NULL. */
int hot_export_groups(int32_t* cell, uint64_t* key, uint32_t* first, uint32_t* count, uint64_t* lpc, uint64_t* lpp,
                      int64_t cap, int64_t* ngroups);
/* accepted cells per sink group by expansion order, last hot_forces / hot_forces_tol; HOST arrays [ngroups], NULL to skip */
int hot_export_group_orders(uint64_t* lmono, uint64_t* lquad, uint64_t* lhexa, int64_t cap, int64_t* ngroups);
/* The interaction lists of ONE sink group as the last hot_forces walked them, as sets
 * (the order inside a list is the walk's and means nothing):
 *   pc_cell [*npc]: indices (ascending-key numbering of hot_export_cells) of the accepted cells,
 *   pc_img  [*npc]: image of each, 25 (nx+2) + 5 (ny+2) + (nz+2), 62 = the box itself (always 62 when open),
 *   pp_body [*npp]: sorted positions (index into key_sorted / perm of hot_export_keys) of the listed bodies;
 *                   the group's OWN bodies in the box itself are not in the list (the kernel pairs them
 *                   separately and skips j = i), so *npp = L_pp - count(group),
 *   pp_img  [*npp]: image of each.
 * HOST arrays; pc_img / pp_img may be NULL; *npc / *npp are always set; HOT_EINVAL if a cap is too small.
 * HOT_EORDER if the group's lists are no longer in the arena (hot_forces ran in several rounds,
 * hot_stats list_chunks > 1, and this group was not in the last one). */
int hot_export_lists(int64_t group, int32_t* pc_cell, uint8_t* pc_img, int64_t pc_cap, int64_t* npc,
                     uint32_t* pp_body, uint8_t* pp_img, int64_t pp_cap, int64_t* npp);
/* moments of the last hot_forces: com [ncells][3] double, m0 [ncells], bmax [ncells] (radius about com
 * holding every body of the cell, PAPER.md:94 / DESIGN.md R-15), m2 [ncells][6] (xx xy xz yy yz zz),
 * m3 [ncells][10], m4 [ncells][15] (degree-major, x>y>z); NULL to skip;
 * m3/m4 only when the last order was 4 (else HOT_EINVAL if requested). */
int hot_export_moments(double* com, float* m0, float* bmax, float* m2, float* m3, float* m4, int64_t cap);
/* hash table: cell index of each key, -1 if absent.  keys, idx: host, [nkeys]. */
int hot_lookup_keys(const uint64_t* keys, int64_t nkeys, int32_t* idx);

#ifdef __cplusplus
}
#endif
#endif /* HOT_H_ */

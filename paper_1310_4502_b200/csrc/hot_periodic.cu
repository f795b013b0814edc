// hot_periodic.cu -- P2/P3: the periodic far field ("sums the infinite series of each
// relevant combination of powers of the co-ordinates ... pre-computed coefficients ... used in a local
// expansion about the center of the volume", p = 8, ws = 2; the uniform background of PAPER.md:76-84).
//
// The 125 explicit image boxes are walked like the box itself (hot_walk.cu / hot_forces.cu).  What is
// left of the periodic Green's function, in units of the box,
//     psi_sm(r) = psi(r) - sum_{|n|_inf <= 2} 1/|r - n|,
//     psi(r)    = sum_n 1/|r - n| - (uniform neutralising background), zero mean over the box,
// is smooth for |r_k| < 3, even in every coordinate, cubic-symmetric, and satisfies
// laplace(psi_sm) = 4 pi (only the background is a source inside the explicit region).  Hence
//     psi_sm(r) = C0 + (2 pi / 3) |r|^2 + c4 K4(r) + c6 K6(r) + c8 K8(r) + O(r^10),
// K_l = the cubic harmonic of degree l (the one harmonic, cube-invariant, homogeneous polynomial of
// degree l, normalised to K_l = x^l + ...).  Four numbers fix the table; they are the Taylor
// coefficients of psi_sm along the x axis, summed here from the Ewald representation of psi
// (axis_coefficient below).
//
// The field of all bodies is then a polynomial of degree 8 in the sink position whose 165
// coefficients are combinations of the 165 global raw moments of the box about its centre:
//     sum_j m_j psi_sm(x - x_j) = sum_g D_g x^g,   D_g = sum_{a >= g} c_a C(a, a-g) (-1)^|a-g| S_(a-g).
// Two kernels: the moments S (one fp64 reduction over the bodies, cached per build) and the
// evaluation of the polynomial and its gradient at every body (fp64; the terms cancel strongly),
// stored per body in fp64 for the interaction kernel to add to its fp64 sums.
// The j = i term stays in: it is the body's own images and background, -m_i xi (SURVEY C-9 step 3).
#include <cmath>
#include <cstring>

#include "hot_internal.h"

#define FAR_P 8
#define FAR_N 165 // multi-indices (a,b,c) with a+b+c <= 8

// position of (a,b,c) in degree-major order, x exponent descending, then y
__host__ __device__ constexpr int fidx(int a, int b, int c) {
    int d = a + b + c;
    return d * (d + 1) * (d + 2) / 6 + (d - a) * (d - a + 1) / 2 + (d - a - b);
}

// ---- host: the coefficient table -------------------------------------------------------------------
namespace {
double g_far_coef[FAR_N];
bool g_far_ready = false;

long double legendre(int l, long double x) {
    long double p0 = 1, p1 = x;
    if (l == 0) return p0;
    for (int k = 2; k <= l; ++k) { long double p = ((2 * k - 1) * x * p1 - (k - 1) * p0) / k; p0 = p1; p1 = p; }
    return p1;
}
// coefficient of x^l (l even, <= 8) in the Taylor series of psi_sm(x, 0, 0), from the Ewald form
//   psi(r) = sum_n erfc(a|r-n|)/|r-n| + (1/pi) sum_{h != 0} exp(-pi^2 h^2/a^2)/h^2 cos(2 pi h.r) - pi/a^2,  a = 2.5
long double axis_coefficient(int l) {
    const long double PI = 3.141592653589793238462643383279502884L, al = 2.5L;
    const int k = l / 2;
    long double fact = 1; for (int i = 2; i <= l; ++i) fact *= i;
    long double kfact = 1; for (int i = 2; i <= k; ++i) kfact *= i;
    // n = 0 real-space term minus its explicit 1/r:  -erf(a x)/x = -(2a/sqrt(pi)) sum_k (-1)^k a^2k x^2k / (k! (2k+1))
    long double co = -(2 * al / sqrtl(PI)) * ((k & 1) ? -1.0L : 1.0L) * powl(al, 2 * k) / (kfact * (2 * k + 1));
    // n != 0 real-space terms: F(x) = G(s), s = |x e_x - n|^2 = s0 + (x^2 - 2 n_x x), G(s) = erfc(a sqrt s)/sqrt s;
    // G^(j)(s0) = E_j / 2^j with E_j = (1/d d/dd)^j [erfc(a d)/d] = (-1)^j B_j,
    // B_0 = erfc(a d)/d, B_j = ((2j-1) B_(j-1) + (2 a^2)^j exp(-a^2 d^2)/(a sqrt(pi))) / d^2   (d = |n|)
    const int NR = 5;
    for (int nx = -NR; nx <= NR; ++nx) for (int ny = -NR; ny <= NR; ++ny) for (int nz = -NR; nz <= NR; ++nz) {
        if (!nx && !ny && !nz) continue;
        const long double d2 = (long double)(nx * nx + ny * ny + nz * nz), d = sqrtl(d2);
        long double B = erfcl(al * d) / d;
        const long double ex = expl(-al * al * d2) / (al * sqrtl(PI));
        long double pw[FAR_P + 1] = {1};             // (x^2 - 2 n_x x)^j as a polynomial in x, truncated at degree 8
        long double acc = l == 0 ? B : 0;            // j = 0 term
        long double jf = 1, two = 1;
        for (int j = 1; j <= l; ++j) {
            B = ((2 * j - 1) * B + powl(2 * al * al, j) * ex) / d2;
            const long double E = (j & 1) ? -B : B;
            long double nw[FAR_P + 1] = {0};         // pw * (x^2 - 2 n_x x)
            for (int e = 0; e <= FAR_P; ++e) {
                if (e + 1 <= FAR_P) nw[e + 1] += -2.0L * nx * pw[e];
                if (e + 2 <= FAR_P) nw[e + 2] += pw[e];
            }
            for (int e = 0; e <= FAR_P; ++e) pw[e] = nw[e];
            jf *= j; two *= 2;
            acc += E / (two * jf) * pw[l];
        }
        co += acc;
    }
    // reciprocal-space sum: d^l/dx^l cos(2 pi h.r) at 0 = (-1)^(l/2) (2 pi h_x)^l
    const int H = 8;
    long double rs = 0;
    for (int hx = -H; hx <= H; ++hx) for (int hy = -H; hy <= H; ++hy) for (int hz = -H; hz <= H; ++hz) {
        const int h2 = hx * hx + hy * hy + hz * hz;
        if (h2 == 0) continue;
        rs += expl(-PI * PI * h2 / (al * al)) / h2 * powl(2 * PI * hx, l);
    }
    co += rs / PI * ((k & 1) ? -1.0L : 1.0L) / fact;
    if (l == 0) co -= PI / (al * al);
    // the 124 explicit neighbour images: 1/|x e_x - n| = sum_l x^l P_l(n_x/|n|) / |n|^(l+1)
    for (int nx = -2; nx <= 2; ++nx) for (int ny = -2; ny <= 2; ++ny) for (int nz = -2; nz <= 2; ++nz) {
        if (!nx && !ny && !nz) continue;
        const long double d = sqrtl((long double)(nx * nx + ny * ny + nz * nz));
        co -= legendre(l, nx / d) / powl(d, l + 1);
    }
    return co;
}
// K_l = x^l + ... : coefficients of the sorted even triples (a >= b >= c) of degree l, from laplace(K_l) = 0
void cubic_harmonic(int l, double (&K)[9][9][9]) {
    int ta[8], tb[8], tc[8], nt = 0;      // sorted even triples of degree l; the first is (l,0,0)
    for (int a = l; a >= 0; a -= 2) for (int b = (l - a < a ? l - a : a); b >= 0; b -= 2) {
        const int c = l - a - b;
        if (c > b || c < 0 || (c & 1)) continue;
        ta[nt] = a; tb[nt] = b; tc[nt] = c; ++nt;
    }
    int ea[8], eb[8], ec[8], ne = 0;      // sorted even triples of degree l-2: one equation each
    for (int a = l - 2; a >= 0; a -= 2) for (int b = (l - 2 - a < a ? l - 2 - a : a); b >= 0; b -= 2) {
        const int c = l - 2 - a - b;
        if (c > b || c < 0 || (c & 1)) continue;
        ea[ne] = a; eb[ne] = b; ec[ne] = c; ++ne;
    }
    auto find = [&](int a, int b, int c) { // index of the sorted version of (a,b,c)
        if (a < b) { int t = a; a = b; b = t; }
        if (b < c) { int t = b; b = c; c = t; }
        if (a < b) { int t = a; a = b; b = t; }
        for (int i = 0; i < nt; ++i) if (ta[i] == a && tb[i] == b && tc[i] == c) return i;
        return -1;
    };
    // A u = rhs with unknowns u_1..u_(nt-1), u_0 = 1
    const int n = nt - 1;
    double A[8][8] = {}, rhs[8] = {};
    for (int e = 0; e < ne; ++e) {
        const int p = ea[e], q = eb[e], r = ec[e];
        const int i1 = find(p + 2, q, r), i2 = find(p, q + 2, r), i3 = find(p, q, r + 2);
        const double w1 = (p + 2.0) * (p + 1.0), w2 = (q + 2.0) * (q + 1.0), w3 = (r + 2.0) * (r + 1.0);
        const int id[3] = {i1, i2, i3}; const double wv[3] = {w1, w2, w3};
        for (int t = 0; t < 3; ++t) { if (id[t] == 0) rhs[e] -= wv[t]; else A[e][id[t] - 1] += wv[t]; }
    }
    for (int c0 = 0; c0 < n; ++c0) { // Gaussian elimination with partial pivoting (n <= 3, ne == n)
        int piv = c0;
        for (int r0 = c0 + 1; r0 < n; ++r0) if (std::fabs(A[r0][c0]) > std::fabs(A[piv][c0])) piv = r0;
        for (int k = 0; k < n; ++k) { double t = A[c0][k]; A[c0][k] = A[piv][k]; A[piv][k] = t; }
        { double t = rhs[c0]; rhs[c0] = rhs[piv]; rhs[piv] = t; }
        for (int r0 = c0 + 1; r0 < n; ++r0) {
            const double f = A[r0][c0] / A[c0][c0];
            for (int k = c0; k < n; ++k) A[r0][k] -= f * A[c0][k];
            rhs[r0] -= f * rhs[c0];
        }
    }
    double u[8] = {1.0};
    for (int r0 = n - 1; r0 >= 0; --r0) {
        double s = rhs[r0];
        for (int k = r0 + 1; k < n; ++k) s -= A[r0][k] * u[k + 1];
        u[r0 + 1] = s / A[r0][r0];
    }
    for (int i = 0; i < nt; ++i) { // spread over all permutations of each triple
        const int p[3] = {ta[i], tb[i], tc[i]};
        const int perm[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};
        for (auto& pm : perm) K[p[pm[0]]][p[pm[1]]][p[pm[2]]] = u[i];
    }
}
void far_build_table() {
    if (g_far_ready) return;
    const double PI = 3.14159265358979323846;
    for (int k = 0; k < FAR_N; ++k) g_far_coef[k] = 0.0;
    g_far_coef[fidx(0, 0, 0)] = (double)axis_coefficient(0);
    g_far_coef[fidx(2, 0, 0)] = g_far_coef[fidx(0, 2, 0)] = g_far_coef[fidx(0, 0, 2)] = 2.0 * PI / 3.0; // the background
    for (int l = 4; l <= FAR_P; l += 2) {
        static double K[9][9][9];
        std::memset(K, 0, sizeof(K));
        cubic_harmonic(l, K);
        const double cl = (double)axis_coefficient(l);
        for (int a = 0; a <= l; a += 2) for (int b = 0; a + b <= l; b += 2) g_far_coef[fidx(a, b, l - a - b)] = cl * K[a][b][l - a - b];
    }
    g_far_ready = true;
}
double binom(int n, int k) { double r = 1; for (int i = 0; i < k; ++i) r = r * (n - i) / (i + 1); return r; }
} // namespace

void far_coefficients(double* out165) { far_build_table(); std::memcpy(out165, g_far_coef, sizeof(g_far_coef)); }

// D_g = sum_{a >= g} c_a C(a, a-g) (-1)^|a-g| S_(a-g)
void far_sink_polynomial(const double* S, double* D) {
    far_build_table();
    for (int k = 0; k < FAR_N; ++k) D[k] = 0.0;
    for (int deg = 0; deg <= FAR_P; deg += 2)
        for (int a = 0; a <= deg; a += 2) for (int b = 0; a + b <= deg; b += 2) {
            const int c = deg - a - b;
            const double co = g_far_coef[fidx(a, b, c)];
            if (co == 0.0) continue;
            for (int i = 0; i <= a; ++i) for (int j = 0; j <= b; ++j) for (int k = 0; k <= c; ++k) { // (i,j,k) = a - g
                const double w = co * binom(a, i) * binom(b, j) * binom(c, k) * (((i + j + k) & 1) ? -1.0 : 1.0);
                D[fidx(a - i, b - j, c - k)] += w * S[fidx(i, j, k)];
            }
        }
}

// ---- device: global raw moments about the box centre, box units -------------------------------------
#define FM_TILE 64
#define FM_THREADS 192 // = 3 * FM_TILE: one thread per (coordinate, body) when the power tables are filled
struct FarIdx { unsigned char a[FAR_N], b[FAR_N], c[FAR_N]; };
__global__ void __launch_bounds__(FM_THREADS) far_moments_kernel(const float4* __restrict__ body, int64_t n, double cx, double cy, double cz,
                                                                 double inv, const __grid_constant__ FarIdx I, double* __restrict__ S) {
    // powers of the three coordinates of a tile of bodies, exponent fastest: the 165 threads read
    // <= 9 consecutive doubles per table (no bank conflicts), threads with equal exponents broadcast.
    // The mass is folded into the x table.
    __shared__ double pw[3][FM_TILE][FAR_P + 1];
    const int t = threadIdx.x;
    const int ma = t < FAR_N ? I.a[t] : 0, mb = t < FAR_N ? I.b[t] : 0, mc = t < FAR_N ? I.c[t] : 0; // this thread's moment
    double acc = 0.0;
    for (int64_t base = (int64_t)blockIdx.x * FM_TILE; base < n; base += (int64_t)gridDim.x * FM_TILE) {
        { // thread t: coordinate k = t / 64 of body t % 64
            const int k = t / FM_TILE, jj = t % FM_TILE;
            const int64_t j = base + jj;
            float4 b = make_float4(0.f, 0.f, 0.f, 0.f);
            if (j < n) b = body[j];
            const double d = k == 0 ? ((double)b.x - cx) * inv : k == 1 ? ((double)b.y - cy) * inv : ((double)b.z - cz) * inv;
            double p = k == 0 ? (j < n ? (double)b.w : 0.0) : 1.0;
#pragma unroll
            for (int e = 0; e <= FAR_P; ++e) { pw[k][jj][e] = p; p *= d; }
        }
        __syncthreads();
        if (t < FAR_N) {
#pragma unroll 8
            for (int j = 0; j < FM_TILE; ++j) acc = fma(pw[0][j][ma] * pw[1][j][mb], pw[2][j][mc], acc);
        }
        __syncthreads();
    }
    if (t < FAR_N) atomicAdd(&S[t], acc);
}

// ---- device: the degree-8 polynomial and its gradient at every body ------------------------------------
struct FarPoly { double D[FAR_N]; };
__global__ void __launch_bounds__(128) far_eval_kernel(const float4* __restrict__ body, int64_t n, double cx, double cy, double cz, double inv,
                                                       const __grid_constant__ FarPoly Q, double* __restrict__ far) {
    __shared__ double D[FAR_N];
    for (int k = threadIdx.x; k < FAR_N; k += blockDim.x) D[k] = Q.D[k];
    __syncthreads();
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 b = body[i];
    const double x = ((double)b.x - cx) * inv, y = ((double)b.y - cy) * inv, z = ((double)b.z - cz) * inv;
    // v = sum_a x^a sum_b y^b sum_c z^c D_abc by nested Horner (z innermost), carrying the partial
    // derivatives along (f' <- f' t + f before f <- f t + c): ~500 fused multiply-adds, no power tables
    double v = 0.0, gx = 0.0, gy = 0.0, gz = 0.0;
#pragma unroll
    for (int a = FAR_P; a >= 0; --a) {
        double B = 0.0, By = 0.0, Bz = 0.0; // sum_b y^b C_ab(z) and its y, z derivatives
#pragma unroll
        for (int bb = FAR_P - a; bb >= 0; --bb) {
            double C = 0.0, Cz = 0.0;       // C_ab(z) = sum_c D_abc z^c and dC/dz
#pragma unroll
            for (int c = FAR_P - a - bb; c >= 0; --c) { Cz = fma(Cz, z, C); C = fma(C, z, D[fidx(a, bb, c)]); }
            By = fma(By, y, B); B = fma(B, y, C); Bz = fma(Bz, y, Cz);
        }
        gx = fma(gx, x, v); v = fma(v, x, B); gy = fma(gy, x, By); gz = fma(gz, x, Bz);
    }
    // a_far = grad / L^2, phi_far = -v / L  (inv = 1/L); kept in fp64, key order: the interaction kernel adds
    // it to its fp64 sums before the one rounding to fp32 (the explicit and the far part cancel strongly)
    double4 r;
    r.x = gx * inv * inv; r.y = gy * inv * inv; r.z = gz * inv * inv; r.w = -v * inv;
    reinterpret_cast<double4*>(far)[i] = r;
}

cudaError_t launch_far_moments(const Tree& t, double* S, cudaStream_t st) {
    FarIdx I;
    for (int d = 0, k = 0; d <= FAR_P; ++d)
        for (int a = d; a >= 0; --a) for (int b = d - a; b >= 0; --b, ++k) { I.a[k] = (unsigned char)a; I.b[k] = (unsigned char)b; I.c[k] = (unsigned char)(d - a - b); }
    cudaError_t e = cudaMemsetAsync(S, 0, sizeof(double) * FAR_N, st);
    if (e != cudaSuccess) return e;
    int64_t nb = (t.n + FM_TILE - 1) / FM_TILE;
    if (nb > 148 * 8) nb = 148 * 8;
    HOT_LAUNCHED(1);
    far_moments_kernel<<<(unsigned)nb, FM_THREADS, 0, st>>>(t.body, t.n, t.lo[0] + 0.5 * t.size, t.lo[1] + 0.5 * t.size, t.lo[2] + 0.5 * t.size,
                                                           1.0 / t.size, I, S);
    return cudaGetLastError();
}
cudaError_t launch_far_eval(const Tree& t, const double* D, double* far, cudaStream_t st) {
    FarPoly Q;
    std::memcpy(Q.D, D, sizeof(Q.D));
    HOT_LAUNCHED(1);
    far_eval_kernel<<<(unsigned)((t.n + 127) / 128), 128, 0, st>>>(t.body, t.n, t.lo[0] + 0.5 * t.size, t.lo[1] + 0.5 * t.size,
                                                                  t.lo[2] + 0.5 * t.size, 1.0 / t.size, Q, far);
    return cudaGetLastError();
}

// ---- fp64 monopoles of the coarse cells (periodic boxes) --------------------------------------------
// A body of a nearly uniform periodic set feels an O(M/L^2) pull towards the centre of the 5^3 explicit
// boxes which the far field cancels to the few-percent-of-that net acceleration; fp32 interaction terms
// carry ~2e-7 of their own size, and the few hundred coarsest cells of the image boxes (levels 0..2, each
// 1/64 of the box mass or more) carry most of that pull.  Their monopole terms are therefore summed here in
// fp64 (25 operations each) and added, with the far field, to the fp64 sums of the interaction kernel, which
// evaluates only their higher moments.  One warp per sink group, two sinks per lane and pass.
#define CM_WARPS 8
__global__ void __launch_bounds__(CM_WARPS * 32) coarse_monopole_kernel(const __grid_constant__ ForceArgs P, const double* __restrict__ far,
                                                                        double* __restrict__ farc, double eps2) {
    __shared__ double4 s_cell[CM_WARPS][32]; // staged coarse cells of a batch: centre (shifted to its image), mass
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    double4* const sc = s_cell[w];
    for (int64_t gi = P.g0 + (int64_t)blockIdx.x * CM_WARPS + w; gi < P.g1; gi += (int64_t)gridDim.x * CM_WARPS) {
        const GroupRec g = P.group[gi];
        const unsigned long long o0 = P.pcoff[gi];
        const int n = (int)P.lpc[gi];
        const uint32_t* const pl = P.pclist + o0;
        const uint8_t* const pi = P.pcimg + o0;
        for (uint32_t s0 = 0; s0 < g.count; s0 += 64) {
            double x[2][3], a[2][4];
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const uint32_t loc = s0 + 32 * i + lane;
                const float4 b = P.body[g.first + (loc < g.count ? loc : 0u)];
                x[i][0] = b.x; x[i][1] = b.y; x[i][2] = b.z;
                a[i][0] = a[i][1] = a[i][2] = a[i][3] = 0.0;
            }
            for (int b0 = 0; b0 < n; b0 += 32) {
                uint32_t e = 0; int im = 62;
                if (b0 + lane < n) { e = pl[b0 + lane]; im = pi[b0 + lane]; }
                const bool coarse = (e & HOT_COARSE_FLAG) != 0;
                const uint32_t m = __ballot_sync(0xffffffffu, coarse);
                if (m == 0) continue;
                if (coarse) {
                    const CellA cA = P.cellA[e & ~HOT_COARSE_FLAG];
                    double4 r;
                    r.x = cA.zx + (double)(im / 25 - 2) * P.size; r.y = cA.zy + (double)((im / 5) % 5 - 2) * P.size;
                    r.z = cA.zz + (double)(im % 5 - 2) * P.size; r.w = (double)cA.m0;
                    sc[__popc(m & ((1u << lane) - 1u))] = r;
                }
                __syncwarp();
                const int nc = __popc(m);
                for (int k = 0; k < nc; ++k) {
                    const double4 c = sc[k];
#pragma unroll
                    for (int i = 0; i < 2; ++i) {
                        const double Rx = x[i][0] - c.x, Ry = x[i][1] - c.y, Rz = x[i][2] - c.z;
                        const double ri = rsqrt(fma(Rx, Rx, fma(Ry, Ry, fma(Rz, Rz, eps2))));
                        const double mr = c.w * ri, mr3 = mr * ri * ri;
                        a[i][0] = fma(-mr3, Rx, a[i][0]); a[i][1] = fma(-mr3, Ry, a[i][1]); a[i][2] = fma(-mr3, Rz, a[i][2]);
                        a[i][3] -= mr;
                    }
                }
                __syncwarp();
            }
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const uint32_t loc = s0 + 32 * i + lane;
                if (loc < g.count) {
                    const double4 f = reinterpret_cast<const double4*>(far)[g.first + loc];
                    double4 r;
                    r.x = f.x + a[i][0]; r.y = f.y + a[i][1]; r.z = f.z + a[i][2]; r.w = f.w + a[i][3];
                    reinterpret_cast<double4*>(farc)[g.first + loc] = r;
                }
            }
        }
    }
}
cudaError_t launch_coarse_monopoles(const ForceArgs& a, const double* far, double* farc, double eps2, cudaStream_t st) {
    const int64_t ng = a.g1 - a.g0;
    if (ng <= 0) return cudaSuccess;
    int64_t nb = (ng + CM_WARPS - 1) / CM_WARPS;
    if (nb > 148 * 16) nb = 148 * 16;
    HOT_LAUNCHED(1);
    coarse_monopole_kernel<<<(unsigned)nb, CM_WARPS * 32, 0, st>>>(a, far, farc, eps2);
    return cudaGetLastError();
}

#!/usr/bin/env python
"""Generator of the high-order (p = 6, 8) particle-cell terms: writes hot_hi_generated.inc.

    python paper_1310_4502_b200/csrc/gen_hi_orders.py          # rewrites the .inc beside this file

PAPER.md:120: "The expression for the force with p=8 in three dimensions begins with 3^8 = 6561 terms.  We resort to
metaprogramming ... producing the necessary interaction routines through p=8 without human intervention."  Here the
"computer algebra" is the multi-index recursion below; no formula is typed by hand beyond eq (5) itself.

Eq (5) with g(R) = (|R|^2 + eps^2)^(-1/2), u = |R|^2 + eps^2:
    d^(n) g contracted with the symmetric moment tensor M^(n) = sum_k c(n,k) D_(n-k)(u) (T^(n,k) . R^(n-2k)),
    T^(n,k) = the k-fold trace of M^(n) (rank m = n - 2k), c(n,k) = n! / (2^k k! m!) pairings,
    D_j = (-1)^j (2j-1)!! u^(-(2j+1)/2),  grad D_j = D_(j+1) R.
    phi_n = -((-1)^n / n!) sum_k c(n,k) D_(n-k) S,              S = T . R^m (full contraction)
    a_n   = +((-1)^n / n!) sum_k c(n,k) [D_(n-k+1) S R + m D_(n-k) V],   V = T . R^(m-1) (a vector), S = V . R.
A symmetric rank-m tensor is indexed by a multi-index beta (|beta| = m, degree-major, x exponent descending, then y):
    S = sum_beta (m!/beta!) T_beta R^beta,   V_i = sum_{|beta'| = m-1} ((m-1)!/beta'!) T_(beta'+e_i) R^beta'.
Scaling (fp32 range): the record holds f_nk T^(n,k) / side^n with f_nk = (-1)^n c(n,k) / n! and side = the cell's side;
with ri = u^(-1/2), rho = R ri, t = side ri:   D_j S = g_j ri t^n (T~ . rho^m),  g_j = (-1)^j (2j-1)!!, so
    phi -= ri   sum_n t^n sum_k g_j S~,        a += ri^2 sum_n t^n sum_k [g_(j+1) S~ rho + m g_j V~],   j = n - k.
Only n = 5 .. P are generated: orders 0-4 are the hand-written kernels of hot_forces.cu.
"""
import os
from math import factorial


def multi(d):
    return [(a, b, d - a - b) for a in range(d, -1, -1) for b in range(d - a, -1, -1)]


def idx_in_degree(beta):
    a, b, c = beta
    d = a + b + c
    return (d - a) * (d - a + 1) // 2 + (d - a - b)


def raw_index(beta):  # position in the degree-major list of all moments (as hot_moments.cu's midx)
    d = sum(beta)
    return d * (d + 1) * (d + 2) // 6 + idx_in_degree(beta)


def dfact(j):  # (2j-1)!!
    r = 1
    for q in range(1, 2 * j, 2):
        r *= q
    return r


def tensors(P):
    """[(n, k, m, offset)] of the record, n = 5..P, and its length."""
    out, off = [], 0
    for n in range(5, P + 1):
        for k in range(0, n // 2 + 1):
            m = n - 2 * k
            if n == 1:
                continue
            out.append((n, k, m, off))
            off += (m + 1) * (m + 2) // 2
    return out, off


def emit(P):
    L = []
    tl, NT = tensors(P)
    L.append(f"// ---- order {P}: {len(tl)} trace tensors, {NT} floats per cell ----")
    L.append(f"template <> struct HiOrder<{P}> {{ static constexpr int NT = {NT}; static constexpr int NRAW = {sum((n + 1) * (n + 2) // 2 for n in range(5, P + 1))}; }};")
    # record builder from raw moments (fp64, unscaled, degree-major through degree P), inv_side = 1 / cell side
    L.append(f"template <> __device__ __forceinline__ void hi_record<{P}>(const double* __restrict__ M, const double inv_side, float* __restrict__ T) {{")
    L.append("    double sc = inv_side * inv_side; sc = sc * sc * inv_side; // inv_side^5")
    for n in range(5, P + 1):
        if n > 5:
            L.append("    sc *= inv_side;")
        for (nn, k, m, off) in tl:
            if nn != n:
                continue
            f = (-1) ** n / (2 ** k * factorial(k) * factorial(m))
            for beta in multi(m):
                terms = []
                for gam in multi(k):
                    w = factorial(k) // (factorial(gam[0]) * factorial(gam[1]) * factorial(gam[2]))
                    src = (beta[0] + 2 * gam[0], beta[1] + 2 * gam[1], beta[2] + 2 * gam[2])
                    terms.append((f"{w}.0 * " if w != 1 else "") + f"M[{raw_index(src)}]")
                L.append(f"    T[{off + idx_in_degree(beta)}] = (float)({f!r} * sc * ({' + '.join(terms)}));")
    L.append("}")
    # evaluation
    L.append("#ifdef HOT_HI_WITH_TERMS // the evaluation routine: only the translation unit of the kernel that calls it (hot_hi.cu)")
    L.append(f"template <> __device__ __noinline__ void hi_terms<{P}>(const float* __restrict__ T, const float rx, const float ry, const float rz, const float ri, const float t,")
    L.append("                                                float& ax, float& ay, float& az, float& ph) {")
    L.append("    // monomials of rho = R ri with their multiplicities d!/beta!, degrees 0 .. P-1")
    names = {}
    L.append("    const float q_0_0 = 1.0f;")
    names[(0, 0, 0)] = "p_0_0_0"
    L.append("    const float p_0_0_0 = 1.0f;")
    for d in range(1, P):
        for beta in multi(d):
            a, b, c = beta
            if a > 0:
                prev, var = (a - 1, b, c), "rx"
            elif b > 0:
                prev, var = (a, b - 1, c), "ry"
            else:
                prev, var = (a, b, c - 1), "rz"
            L.append(f"    const float p_{a}_{b}_{c} = p_{prev[0]}_{prev[1]}_{prev[2]} * {var};")
    def q(beta):  # monomial with multiplicity
        d = sum(beta)
        w = factorial(d) // (factorial(beta[0]) * factorial(beta[1]) * factorial(beta[2]))
        return (f"{float(w)!r}f * " if w != 1 else "") + f"p_{beta[0]}_{beta[1]}_{beta[2]}"
    L.append("    float sphi = 0.0f, sr = 0.0f, svx = 0.0f, svy = 0.0f, svz = 0.0f; // sums over n of t^n x (potential, coefficient of rho, vector part)")
    L.append("    float tn = t * t; tn = tn * tn * t; // t^5")
    for n in range(5, P + 1):
        if n > 5:
            L.append("    tn *= t;")
        L.append(f"    {{ // n = {n}")
        L.append("        float nphi = 0.0f, nr = 0.0f, nvx = 0.0f, nvy = 0.0f, nvz = 0.0f;")
        for (nn, k, m, off) in tl:
            if nn != n:
                continue
            j = n - k
            gj = float((-1) ** j * dfact(j))
            gj1 = float((-1) ** (j + 1) * dfact(j + 1))
            if m == 0:
                L.append(f"        {{ const float S = T[{off}]; nphi = fmaf({gj!r}f, S, nphi); nr = fmaf({gj1!r}f, S, nr); }} // (n,k) = ({n},{k}): scalar trace")
                continue
            L.append(f"        {{ // (n,k) = ({n},{k}): rank {m}, D index {j}")
            L.append("            float vx = 0.0f, vy = 0.0f, vz = 0.0f;")
            for bp in multi(m - 1):
                ix = off + idx_in_degree((bp[0] + 1, bp[1], bp[2]))
                iy = off + idx_in_degree((bp[0], bp[1] + 1, bp[2]))
                iz = off + idx_in_degree((bp[0], bp[1], bp[2] + 1))
                L.append(f"            {{ const float w = {q(bp)}; vx = fmaf(T[{ix}], w, vx); vy = fmaf(T[{iy}], w, vy); vz = fmaf(T[{iz}], w, vz); }}")
            L.append("            const float S = fmaf(vx, rx, fmaf(vy, ry, vz * rz));")
            L.append(f"            nphi = fmaf({gj!r}f, S, nphi); nr = fmaf({gj1!r}f, S, nr);")
            L.append(f"            nvx = fmaf({float(m) * gj!r}f, vx, nvx); nvy = fmaf({float(m) * gj!r}f, vy, nvy); nvz = fmaf({float(m) * gj!r}f, vz, nvz);")
            L.append("        }")
        L.append("        sphi = fmaf(tn, nphi, sphi); sr = fmaf(tn, nr, sr); svx = fmaf(tn, nvx, svx); svy = fmaf(tn, nvy, svy); svz = fmaf(tn, nvz, svz);")
        L.append("    }")
    L.append("    const float ri2 = ri * ri;")
    L.append("    ph = fmaf(-ri, sphi, ph);")
    L.append("    ax = fmaf(ri2, fmaf(sr, rx, svx), ax); ay = fmaf(ri2, fmaf(sr, ry, svy), ay); az = fmaf(ri2, fmaf(sr, rz, svz), az);")
    L.append("}")
    L.append("#endif")
    return L


def generate():
    L = ["// GENERATED by gen_hi_orders.py -- do not edit; regenerate with `python paper_1310_4502_b200/csrc/gen_hi_orders.py`.",
         "// High-order (n = 5 .. P, P = 6, 8) terms of eq (5) (PAPER.md:104-107, 120); the derivation is in the generator's docstring.",
         "template <int P> struct HiOrder;",
         "template <int P> __device__ __forceinline__ void hi_record(const double* __restrict__ M, const double inv_side, float* __restrict__ T);",
         "template <int P> __device__ __noinline__ void hi_terms(const float* __restrict__ T, const float rx, const float ry, const float rz, const float ri, const float t,",
         "                                           float& ax, float& ay, float& az, float& ph);"]
    for P in (6, 8):
        L += emit(P)
    return "\n".join(L) + "\n"


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "hot_hi_generated.inc")
    open(path, "w").write(generate())
    print(path, len(generate().splitlines()), "lines")

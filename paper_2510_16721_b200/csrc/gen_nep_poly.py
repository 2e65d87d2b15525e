"""Writes nep_poly.cuh: the 35 monomials x^a y^b z^c of degree <= 4 (the independent components of the symmetric
tensors u^(x)l, l = 0..4), their multiplicities in the Frobenius norm, and the value / gradient of a polynomial
sum_c C_c m_c(u).  Run from this directory:  python gen_nep_poly.py > nep_poly.cuh
Order of the components: degree by degree; within a degree a >= ... as listed in EXPS."""
from math import factorial

EXPS = []
for deg in range(5):
    for a in range(deg, -1, -1):
        for b in range(deg - a, -1, -1):
            EXPS.append((a, b, deg - a - b))


def mult(e):
    return factorial(sum(e)) // (factorial(e[0]) * factorial(e[1]) * factorial(e[2]))


def main():
    n = len(EXPS)
    idx = {e: i for i, e in enumerate(EXPS)}
    out = []
    out.append("// nep_poly.cuh -- written by gen_nep_poly.py (do not edit): monomials of degree <= 4 in the unit vector u.")
    out.append("// component c <-> exponents (a, b, c) of x^a y^b z^c; kNepMult = multiplicity of the component in |u^(x)l|^2.")
    out.append("#pragma once")
    out.append("namespace cfn {")
    out.append("constexpr int kNepC = %d;  // 1 + 3 + 6 + 10 + 15" % n)
    out.append("constexpr int kNepDegStart[6] = {0, 1, 4, 10, 20, 35};")
    out.append("__device__ __constant__ double kNepMult[kNepC] = {%s};" % ", ".join("%d.0" % mult(e) for e in EXPS))
    out.append("// exponents: " + " ".join("%d:%d%d%d" % (i, *e) for i, e in enumerate(EXPS)))
    out.append("__device__ __forceinline__ void nep_monomials(double x, double y, double z, double (&m)[kNepC]) {")
    out.append("    m[0] = 1.0;")
    for i, e in enumerate(EXPS):
        if i == 0:
            continue
        # m[e] = m[e - unit] * var, using the first variable with a positive exponent
        if e[0] > 0:
            p, v = (e[0] - 1, e[1], e[2]), "x"
        elif e[1] > 0:
            p, v = (e[0], e[1] - 1, e[2]), "y"
        else:
            p, v = (e[0], e[1], e[2] - 1), "z"
        out.append("    m[%d] = m[%d] * %s;" % (i, idx[p], v))
    out.append("}")
    out.append("// Gradient of phi(u) = sum_c C_c m_c(u), degree by degree: g[l-1] = grad of the degree-l part, l = 1..4, from")
    out.append("// the monomials of degree <= 3.  (Euler: u . g[l-1] = l phi_l, so the value follows from the gradients.)")
    out.append("__device__ __forceinline__ void nep_poly_grad(const double (&C)[kNepC], const double (&m)[kNepC], double (&g)[4][3]) {")
    for deg in range(1, 5):
        for var in range(3):
            terms = []
            for i, e in enumerate(EXPS):
                if sum(e) != deg or e[var] == 0:
                    continue
                p = list(e)
                p[var] -= 1
                k = e[var]
                terms.append("%sC[%d] * m[%d]" % ("" if k == 1 else "%d.0 * " % k, i, idx[tuple(p)]))
            out.append("    g[%d][%d] = %s;" % (deg - 1, var, " + ".join(terms)))
    out.append("}")
    out.append("}  // namespace cfn")
    print("\n".join(out))


if __name__ == "__main__":
    main()

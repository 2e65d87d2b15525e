// nep_poly.cuh -- written by gen_nep_poly.py (do not edit): monomials of degree <= 4 in the unit vector u.
// component c <-> exponents (a, b, c) of x^a y^b z^c; kNepMult = multiplicity of the component in |u^(x)l|^2.
#pragma once
namespace cfn {
constexpr int kNepC = 35;  // 1 + 3 + 6 + 10 + 15
constexpr int kNepDegStart[6] = {0, 1, 4, 10, 20, 35};
__device__ __constant__ double kNepMult[kNepC] = {1.0, 1.0, 1.0, 1.0, 1.0, 2.0, 2.0, 1.0, 2.0, 1.0, 1.0, 3.0, 3.0, 3.0, 6.0, 3.0, 1.0, 3.0, 3.0, 1.0, 1.0, 4.0, 4.0, 6.0, 12.0, 6.0, 4.0, 12.0, 12.0, 4.0, 1.0, 4.0, 6.0, 4.0, 1.0};
// exponents: 0:000 1:100 2:010 3:001 4:200 5:110 6:101 7:020 8:011 9:002 10:300 11:210 12:201 13:120 14:111 15:102 16:030 17:021 18:012 19:003 20:400 21:310 22:301 23:220 24:211 25:202 26:130 27:121 28:112 29:103 30:040 31:031 32:022 33:013 34:004
__device__ __forceinline__ void nep_monomials(double x, double y, double z, double (&m)[kNepC]) {
    m[0] = 1.0;
    m[1] = m[0] * x;
    m[2] = m[0] * y;
    m[3] = m[0] * z;
    m[4] = m[1] * x;
    m[5] = m[2] * x;
    m[6] = m[3] * x;
    m[7] = m[2] * y;
    m[8] = m[3] * y;
    m[9] = m[3] * z;
    m[10] = m[4] * x;
    m[11] = m[5] * x;
    m[12] = m[6] * x;
    m[13] = m[7] * x;
    m[14] = m[8] * x;
    m[15] = m[9] * x;
    m[16] = m[7] * y;
    m[17] = m[8] * y;
    m[18] = m[9] * y;
    m[19] = m[9] * z;
    m[20] = m[10] * x;
    m[21] = m[11] * x;
    m[22] = m[12] * x;
    m[23] = m[13] * x;
    m[24] = m[14] * x;
    m[25] = m[15] * x;
    m[26] = m[16] * x;
    m[27] = m[17] * x;
    m[28] = m[18] * x;
    m[29] = m[19] * x;
    m[30] = m[16] * y;
    m[31] = m[17] * y;
    m[32] = m[18] * y;
    m[33] = m[19] * y;
    m[34] = m[19] * z;
}
// Gradient of phi(u) = sum_c C_c m_c(u), degree by degree: g[l-1] = grad of the degree-l part, l = 1..4, from
// the monomials of degree <= 3.  (Euler: u . g[l-1] = l phi_l, so the value follows from the gradients.)
__device__ __forceinline__ void nep_poly_grad(const double (&C)[kNepC], const double (&m)[kNepC], double (&g)[4][3]) {
    g[0][0] = C[1] * m[0];
    g[0][1] = C[2] * m[0];
    g[0][2] = C[3] * m[0];
    g[1][0] = 2.0 * C[4] * m[1] + C[5] * m[2] + C[6] * m[3];
    g[1][1] = C[5] * m[1] + 2.0 * C[7] * m[2] + C[8] * m[3];
    g[1][2] = C[6] * m[1] + C[8] * m[2] + 2.0 * C[9] * m[3];
    g[2][0] = 3.0 * C[10] * m[4] + 2.0 * C[11] * m[5] + 2.0 * C[12] * m[6] + C[13] * m[7] + C[14] * m[8] + C[15] * m[9];
    g[2][1] = C[11] * m[4] + 2.0 * C[13] * m[5] + C[14] * m[6] + 3.0 * C[16] * m[7] + 2.0 * C[17] * m[8] + C[18] * m[9];
    g[2][2] = C[12] * m[4] + C[14] * m[5] + 2.0 * C[15] * m[6] + C[17] * m[7] + 2.0 * C[18] * m[8] + 3.0 * C[19] * m[9];
    g[3][0] = 4.0 * C[20] * m[10] + 3.0 * C[21] * m[11] + 3.0 * C[22] * m[12] + 2.0 * C[23] * m[13] + 2.0 * C[24] * m[14] + 2.0 * C[25] * m[15] + C[26] * m[16] + C[27] * m[17] + C[28] * m[18] + C[29] * m[19];
    g[3][1] = C[21] * m[10] + 2.0 * C[23] * m[11] + C[24] * m[12] + 3.0 * C[26] * m[13] + 2.0 * C[27] * m[14] + C[28] * m[15] + 4.0 * C[30] * m[16] + 3.0 * C[31] * m[17] + 2.0 * C[32] * m[18] + C[33] * m[19];
    g[3][2] = C[22] * m[10] + C[24] * m[11] + 2.0 * C[25] * m[12] + C[27] * m[13] + 2.0 * C[28] * m[14] + 3.0 * C[29] * m[15] + C[31] * m[16] + 2.0 * C[32] * m[17] + 3.0 * C[33] * m[18] + 4.0 * C[34] * m[19];
}
}  // namespace cfn

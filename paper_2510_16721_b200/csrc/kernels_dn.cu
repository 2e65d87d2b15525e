// kernels_dn.cu -- K2, pass 1, for the descriptor-network potential CFNEB_POT_DNN (include/cfneb.h): a potential of
// the SHAPE of the paper's NEP (radial and angular descriptors of an atom's environment fed to a small
// network), with seeded weights because the trained ones are not available.  Like
// any potential of that class it enters the path only through the partial forces p^ij = dU_i/dr^ij of Eq. 5; pass 2
// (f^ij = p^ij - p^ji, F_i, virial of Eq. 8) is the kernel the Stillinger-Weber potential uses (kernels_sw.cu).
//   f_k(r)  = 1/2 [T_k(x) + 1] fc(r),  x = 2 (r/r_c - 1)^2 - 1,  fc = 1/2 [1 + cos(pi r/r_c)]
//   q_k     = sum_j f_k(r_ij)                                                   k < K
//   q_{nl}  = sum_j sum_k f_n(r_ij) f_n(r_ik) P_l(cos theta_jik)                 n < M, l = 1..L
//   U_i     = sum_mu W1_mu tanh(sum_d W0_{mu d} q_d - b0_mu)
//   p^ij    = sum_d (dU_i/dq_d) dq_d/dr^ij
// The double sum over the environment is never formed.  With u = r/|r| and the moments of the environment
//   S^(l)_n = sum_j f_n(r_ij) u_ij^(x)l      (l = 0..3: 1 + 3 + 6 + 10 = 20 independent components per n)
// the powers of cos theta_jik = u_ij . u_ik factorise, sum_jk f f cos^l = |S^(l)|^2 (Frobenius norm), so
//   q_{n1} = |S1|^2,  q_{n2} = 3/2 |S2|^2 - 1/2 S0^2,  q_{n3} = 5/2 |S3|^2 - 3/2 |S1|^2,  q_k = S0_k
// and both the descriptors and the partial forces are linear-time in the number of neighbours.  One thread per atom
// walks its list twice: first the 80 moments (registers), then -- after the network and dU/dS^(l)_n, which overwrite
// the moments in place -- one partial force per list entry from the polynomial phi_n(u) = sum_c (dU/dS_nc) u^c:
//   p^ij = sum_n [ f_n'(r) phi_n(u) u + f_n(r)/r (I - u u^T) grad_u phi_n(u) ].
// No per-thread environment array, hence no limit on the atoms inside the cut-off other than the list capacity.
#include "cfneb_internal.cuh"
#include "trig01.cuh"

namespace cfn {

constexpr int kDnK = 4, kDnL = 3, kDnC = 20;  // radial functions, angular orders, moment components per function

// multiplicity of each independent component in the Frobenius norm of the symmetric tensors
// order: 1 | x y z | xx yy zz xy xz yz | xxx yyy zzz xxy xxz yyx yyz zzx zzy xyz
__device__ __forceinline__ void dn_monomials(double x, double y, double z, double (&m)[kDnC]) {
    m[0] = 1.0; m[1] = x; m[2] = y; m[3] = z;
    m[4] = x * x; m[5] = y * y; m[6] = z * z; m[7] = x * y; m[8] = x * z; m[9] = y * z;
    m[10] = m[4] * x; m[11] = m[5] * y; m[12] = m[6] * z; m[13] = m[4] * y; m[14] = m[4] * z;
    m[15] = m[5] * x; m[16] = m[5] * z; m[17] = m[6] * x; m[18] = m[6] * y; m[19] = m[7] * z;
}

// radial basis and its derivative with respect to r; t = r / r_c
__device__ __forceinline__ void dn_basis(double t, double irc, double (&f)[kDnK], double (&df)[kDnK]) {
    double sn, cs;
    sincospi01(t, sn, cs);  // 0 < t < 1 inside the cut-off
    const double fc = 0.5 + 0.5 * cs, dfc = -0.5 * sn * (3.14159265358979323846 * irc);
    const double x = 2.0 * (t - 1.0) * (t - 1.0) - 1.0, dx_dr = 4.0 * (t - 1.0) * irc;
    const double T[kDnK] = {1.0, x, 2.0 * x * x - 1.0, (4.0 * x * x - 3.0) * x};  // Chebyshev, closed forms
    const double dT[kDnK] = {0.0, 1.0, 4.0 * x, 12.0 * x * x - 3.0};
#pragma unroll
    for (int k = 0; k < kDnK; ++k) {
        const double g = 0.5 * (T[k] + 1.0);
        f[k] = g * fc;
        df[k] = 0.5 * dT[k] * dx_dr * fc + g * dfc;
    }
}

// MT = number of radial functions with angular channels (pot[2]): the moments of order 1..3 of the others are never
// formed, which frees their registers.
template <int MT>
__global__ void __launch_bounds__(kThreadsAtom, 2) dn_partial_kernel(Dev d, int p_lo) {
    int p;
    if (!image_of(blockIdx.y, p_lo, d.ctl->P, p)) return;
    const int slot = d.order[p];
    __shared__ double sh[9];
    __shared__ double red[64];
    __shared__ double sW[kDnWeights];
    const int K = (int)d.pot[1], M = MT, L = (int)d.pot[3], H = (int)d.pot[4], D = K + M * L;
    if (threadIdx.x < 9) sh[threadIdx.x] = d.geom[slot].h[threadIdx.x];
    for (int t = threadIdx.x; t < H * D + 2 * H; t += blockDim.x) sW[t] = d.dn_w[t];
    __syncthreads();
    const double *W0 = sW, *b0 = sW + H * D, *W1 = sW + H * D + H;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = i < d.N;
    const double rc = d.r_cut, rc2 = rc * rc, irc = 1.0 / rc;
    double ui[1] = {0.0};
    if (valid) {
        const double4 *Rc = d.Rc + (size_t)slot * d.Npad;
        const uint32_t *lp = d.nbr_list + (size_t)slot * d.cap * d.Npad + i;
        double *part = d.part + (size_t)slot * d.cap * 3 * d.Npad + i;  // part[(k * 3 + m) * Npad]
        const double4 ri = Rc[i];
        const int cnt = live_rows(d, slot, i);  // rows past it cannot be in range and are neither written nor read
        // the list walk is software-pipelined: entry k + 2 and the coordinates of entry k + 1 are in flight while
        // entry k is evaluated (the list has 16 rows of slack behind the last one; index 0 is a valid atom)
        uint32_t e_nn;
        double4 rj_n;
        uint32_t e_n;
        auto walk_begin = [&]() {
            e_n = lp[0];
            e_nn = lp[(size_t)d.Npad];
            rj_n = Rc[e_n & kIdxMask];
        };
        auto pair_vec = [&](int k, double &dx, double &dy, double &dz) {
            const uint32_t code = e_n >> kShiftBits;
            const double4 rj = rj_n;
            e_n = e_nn;
            e_nn = lp[(size_t)(k + 2) * d.Npad];
            rj_n = Rc[e_n & kIdxMask];
            dx = rj.x - ri.x; dy = rj.y - ri.y; dz = rj.z - ri.z;
            if (code != kCodeCenter) {
                const double n0 = (double)((int)(code & 7u) - 4), n1 = (double)((int)((code >> 3) & 7u) - 4),
                             n2 = (double)((int)((code >> 6) & 7u) - 4);
                dx += n0 * sh[0] + n1 * sh[3] + n2 * sh[6];
                dy += n0 * sh[1] + n1 * sh[4] + n2 * sh[7];
                dz += n0 * sh[2] + n1 * sh[5] + n2 * sh[8];
            }
            return dx * dx + dy * dy + dz * dz;
        };
        // walk 1: moments S[n][c] = sum_j f_n(r_ij) u_ij^c
        double S[kDnK][kDnC];
#pragma unroll
        for (int n = 0; n < kDnK; ++n)
#pragma unroll
            for (int c = 0; c < kDnC; ++c) S[n][c] = 0.0;
        walk_begin();
        for (int k = 0; k < cnt; ++k) {
            double dx, dy, dz;
            const double r2 = pair_vec(k, dx, dy, dz);
            if (!(r2 < rc2)) continue;
            const double inv = rsqrt(r2), r = r2 * inv;
            double f[kDnK], df[kDnK], m[kDnC];
            dn_basis(r * irc, irc, f, df);
            dn_monomials(dx * inv, dy * inv, dz * inv, m);
#pragma unroll
            for (int n = 0; n < kDnK; ++n)
#pragma unroll
                for (int c = 0; c < kDnC; ++c)
                    if (c == 0 || n < MT) S[n][c] += f[n] * m[c];
        }
        // descriptors of the angular channels (dense [n][l]; the radial ones are S[k][0])
        double qa[kDnK][kDnL] = {};
#pragma unroll
        for (int n = 0; n < MT; ++n) {
            const double s1 = S[n][1] * S[n][1] + S[n][2] * S[n][2] + S[n][3] * S[n][3];
            const double s2 = S[n][4] * S[n][4] + S[n][5] * S[n][5] + S[n][6] * S[n][6] +
                              2.0 * (S[n][7] * S[n][7] + S[n][8] * S[n][8] + S[n][9] * S[n][9]);
            const double s3 = S[n][10] * S[n][10] + S[n][11] * S[n][11] + S[n][12] * S[n][12] +
                              3.0 * (S[n][13] * S[n][13] + S[n][14] * S[n][14] + S[n][15] * S[n][15] + S[n][16] * S[n][16] +
                                     S[n][17] * S[n][17] + S[n][18] * S[n][18]) +
                              6.0 * S[n][19] * S[n][19];
            qa[n][0] = s1;
            qa[n][1] = 1.5 * s2 - 0.5 * S[n][0] * S[n][0];
            qa[n][2] = 2.5 * s3 - 1.5 * s1;
        }
        // network forward, and its gradient with respect to the descriptors (Fr radial, Fa angular)
        double Fr[kDnK] = {0.0, 0.0, 0.0, 0.0}, Fa[kDnK][kDnL];
#pragma unroll
        for (int n = 0; n < kDnK; ++n)
#pragma unroll
            for (int l = 0; l < kDnL; ++l) Fa[n][l] = 0.0;
        for (int mu = 0; mu < H; ++mu) {
            const double *w = W0 + mu * D;
            double z = -b0[mu];
#pragma unroll
            for (int k = 0; k < kDnK; ++k)
                if (k < K) z += w[k] * S[k][0];
#pragma unroll
            for (int n = 0; n < kDnK; ++n)
#pragma unroll
                for (int l = 0; l < kDnL; ++l)
                    if (n < M && l < L) z += w[K + n * L + l] * qa[n][l];
            const double th = tanh(z), g = W1[mu] * (1.0 - th * th);
            ui[0] += W1[mu] * th;
#pragma unroll
            for (int k = 0; k < kDnK; ++k)
                if (k < K) Fr[k] += g * w[k];
#pragma unroll
            for (int n = 0; n < kDnK; ++n)
#pragma unroll
                for (int l = 0; l < kDnL; ++l)
                    if (n < M && l < L) Fa[n][l] += g * w[K + n * L + l];
        }
        // dU/dS, in place: S[n][c] := G[n][c]
#pragma unroll
        for (int n = 0; n < kDnK; ++n) {
            S[n][0] = Fr[n] - Fa[n][1] * S[n][0];
            if (n >= MT) continue;
            const double g1 = 2.0 * Fa[n][0] - 3.0 * Fa[n][2], g2 = 3.0 * Fa[n][1], g3 = 5.0 * Fa[n][2];
#pragma unroll
            for (int c = 1; c < 4; ++c) S[n][c] *= g1;
#pragma unroll
            for (int c = 4; c < 7; ++c) S[n][c] *= g2;
#pragma unroll
            for (int c = 7; c < 10; ++c) S[n][c] *= 2.0 * g2;
#pragma unroll
            for (int c = 10; c < 13; ++c) S[n][c] *= g3;
#pragma unroll
            for (int c = 13; c < 19; ++c) S[n][c] *= 3.0 * g3;
            S[n][19] *= 6.0 * g3;
        }
        // walk 2: one partial force per list entry (zero outside the cut-off)
        walk_begin();
        for (int k = 0; k < cnt; ++k) {
            double dx, dy, dz;
            const double r2 = pair_vec(k, dx, dy, dz);
            double px = 0.0, py = 0.0, pz = 0.0;
            if (r2 < rc2) {
                const double inv = rsqrt(r2), r = r2 * inv;
                const double x = dx * inv, y = dy * inv, z = dz * inv;
                double f[kDnK], df[kDnK], m[kDnC];
                dn_basis(r * irc, irc, f, df);
                dn_monomials(x, y, z, m);
                double C[kDnC], dphi = 0.0;  // C = sum_n f_n G_n (coefficients of phi), dphi = sum_n f_n' phi_n(u)
#pragma unroll
                for (int c = 0; c < kDnC; ++c) {
                    double cc = 0.0, dc = 0.0;
#pragma unroll
                    for (int n = 0; n < kDnK; ++n)
                        if (c == 0 || n < MT) { cc += f[n] * S[n][c]; dc += df[n] * S[n][c]; }
                    C[c] = cc;
                    dphi += dc * m[c];
                }
                const double gx = C[1] + 2.0 * C[4] * x + C[7] * y + C[8] * z + 3.0 * C[10] * m[4] + 2.0 * C[13] * m[7] +
                                  2.0 * C[14] * m[8] + C[15] * m[5] + C[17] * m[6] + C[19] * m[9];
                const double gy = C[2] + 2.0 * C[5] * y + C[7] * x + C[9] * z + 3.0 * C[11] * m[5] + C[13] * m[4] +
                                  2.0 * C[15] * m[7] + 2.0 * C[16] * m[9] + C[18] * m[6] + C[19] * m[8];
                const double gz = C[3] + 2.0 * C[6] * z + C[8] * x + C[9] * y + 3.0 * C[12] * m[6] + C[14] * m[4] +
                                  C[16] * m[5] + 2.0 * C[17] * m[8] + 2.0 * C[18] * m[9] + C[19] * m[7];
                const double ug = x * gx + y * gy + z * gz;
                px = dphi * x + inv * (gx - ug * x);
                py = dphi * y + inv * (gy - ug * y);
                pz = dphi * z + inv * (gz - ug * z);
            }
            part[(size_t)(k * 3 + 0) * d.Npad] = px;
            part[(size_t)(k * 3 + 1) * d.Npad] = py;
            part[(size_t)(k * 3 + 2) * d.Npad] = pz;
        }
    }
    double ui_lo = 0.0;
    block_sum_dd(ui[0], ui_lo, red);
    if (threadIdx.x == 0) {
        double *out = d.part_force + ((size_t)slot * d.nblk_force + blockIdx.x) * kNForcePart;
        out[7] = ui[0];
        out[9] = ui_lo;
    }
}

void launch_force_dn(const Dev &d, int p_lo, cudaStream_t st) {
    const int nimg = images_in_grid(d.S, p_lo);
    if (nimg <= 0) return;
    dim3 grid(d.nblk_atom, nimg);
    switch ((int)d.pot[2]) {
        case 1: dn_partial_kernel<1><<<grid, kThreadsAtom, 0, st>>>(d, p_lo); break;
        case 2: dn_partial_kernel<2><<<grid, kThreadsAtom, 0, st>>>(d, p_lo); break;
        case 3: dn_partial_kernel<3><<<grid, kThreadsAtom, 0, st>>>(d, p_lo); break;
        default: dn_partial_kernel<4><<<grid, kThreadsAtom, 0, st>>>(d, p_lo); break;
    }
    launch_pair_forces_manybody(d, p_lo, st);
}

}  // namespace cfn

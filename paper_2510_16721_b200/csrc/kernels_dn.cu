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
// One thread per atom: gather the in-range environment (<= 32 neighbours), descriptors, network forward and its
// gradient with respect to the descriptors, then one sweep over the pairs of the environment for the partial forces.
// The pair sums run over j < k and are doubled (the summand is symmetric); the j = k terms (cos = 1, P_l = 1) are
// added separately.  Weights sit in shared memory, the per-thread environment in local memory.
#include "cfneb_internal.cuh"

namespace cfn {

constexpr int kDnEnv = 32, kDnK = 4, kDnD = 16, kDnH = 8;

__global__ void __launch_bounds__(kThreadsAtom) dn_partial_kernel(Dev d, int p_lo) {
    int p;
    if (!image_of(blockIdx.y, p_lo, d.ctl->P, p)) return;
    const int slot = d.order[p];
    __shared__ double sh[9];
    __shared__ double red[32];
    __shared__ double sW[kDnWeights];
    const int K = (int)d.pot[1], M = (int)d.pot[2], L = (int)d.pot[3], H = (int)d.pot[4], D = K + M * L;
    const int nk = K > M ? K : M;
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
        const int cnt = d.nbr_count[(size_t)slot * d.Npad + i];
        double ux[kDnEnv], uy[kDnEnv], uz[kDnEnv], ir[kDnEnv];          // unit vectors and 1/r
        double f[kDnK][kDnEnv], df[kDnK][kDnEnv];
        double px[kDnEnv], py[kDnEnv], pz[kDnEnv];
        int ek[kDnEnv];
        int n = 0;
        bool overflow = false;
        for (int k = 0; k < cnt; ++k) {
            const uint32_t e = lp[(size_t)k * d.Npad];
            const uint32_t code = e >> kShiftBits;
            const double4 rj = Rc[e & kIdxMask];
            double dx = rj.x - ri.x, dy = rj.y - ri.y, dz = rj.z - ri.z;
            if (code != kCodeCenter) {
                const double n0 = (double)((int)(code & 7u) - 4), n1 = (double)((int)((code >> 3) & 7u) - 4),
                             n2 = (double)((int)((code >> 6) & 7u) - 4);
                dx += n0 * sh[0] + n1 * sh[3] + n2 * sh[6];
                dy += n0 * sh[1] + n1 * sh[4] + n2 * sh[7];
                dz += n0 * sh[2] + n1 * sh[5] + n2 * sh[8];
            }
            const double r2 = dx * dx + dy * dy + dz * dz;
            if (!(r2 < rc2)) continue;
            if (n >= kDnEnv) { overflow = true; continue; }
            const double r = sqrt(r2), inv = 1.0 / r, t = r * irc;
            ux[n] = dx * inv; uy[n] = dy * inv; uz[n] = dz * inv; ir[n] = inv; ek[n] = k;
            double sn, cs;
            sincospi(t, &sn, &cs);
            const double fc = 0.5 + 0.5 * cs, dfc = -0.5 * sn * (3.14159265358979323846 * irc);
            const double x = 2.0 * (t - 1.0) * (t - 1.0) - 1.0, dx_dr = 4.0 * (t - 1.0) * irc;
            // Chebyshev polynomials T_0..T_3 and their derivatives, closed forms
            const double T[kDnK] = {1.0, x, 2.0 * x * x - 1.0, (4.0 * x * x - 3.0) * x};
            const double dT[kDnK] = {0.0, 1.0, 4.0 * x, 12.0 * x * x - 3.0};
#pragma unroll
            for (int k2 = 0; k2 < kDnK; ++k2) {
                const double g = 0.5 * (T[k2] + 1.0);
                f[k2][n] = k2 < nk ? g * fc : 0.0;
                df[k2][n] = k2 < nk ? 0.5 * dT[k2] * dx_dr * fc + g * dfc : 0.0;
            }
            ++n;
        }
        if (overflow) set_error(d.ctl, CFNEB_ENEIGH_OVERFLOW);

        // descriptors
        double q[kDnD];
#pragma unroll
        for (int t = 0; t < kDnD; ++t) q[t] = 0.0;
        for (int a = 0; a < n; ++a) {
            for (int k = 0; k < K; ++k) q[k] += f[k][a];
            for (int m = 0; m < M; ++m) {
                const double w = f[m][a] * f[m][a];
                for (int l = 0; l < L; ++l) q[K + m * L + l] += w;  // j = k: P_l(1) = 1
            }
            for (int b = a + 1; b < n; ++b) {
                const double c = ux[a] * ux[b] + uy[a] * uy[b] + uz[a] * uz[b];
                const double P[3] = {c, 1.5 * c * c - 0.5, (2.5 * c * c - 1.5) * c};
                for (int m = 0; m < M; ++m) {
                    const double w = 2.0 * f[m][a] * f[m][b];
                    for (int l = 0; l < L; ++l) q[K + m * L + l] += w * P[l];
                }
            }
        }
        // network forward and dU/dq
        double Fd[kDnD];
#pragma unroll
        for (int t = 0; t < kDnD; ++t) Fd[t] = 0.0;
        for (int mu = 0; mu < H; ++mu) {
            double z = -b0[mu];
            for (int t = 0; t < D; ++t) z += W0[mu * D + t] * q[t];
            const double th = tanh(z), g = W1[mu] * (1.0 - th * th);
            ui[0] += W1[mu] * th;
            for (int t = 0; t < D; ++t) Fd[t] += g * W0[mu * D + t];
        }
        // partial forces
        for (int a = 0; a < n; ++a) {
            double g = 0.0;
            for (int k = 0; k < K; ++k) g += Fd[k] * df[k][a];
            for (int m = 0; m < M; ++m) {
                double s = 0.0;
                for (int l = 0; l < L; ++l) s += Fd[K + m * L + l];
                g += 2.0 * df[m][a] * f[m][a] * s;
            }
            px[a] = g * ux[a]; py[a] = g * uy[a]; pz[a] = g * uz[a];
        }
        for (int a = 0; a < n; ++a)
            for (int b = a + 1; b < n; ++b) {
                const double c = ux[a] * ux[b] + uy[a] * uy[b] + uz[a] * uz[b];
                const double P[3] = {c, 1.5 * c * c - 0.5, (2.5 * c * c - 1.5) * c};
                const double dP[3] = {1.0, 3.0 * c, 7.5 * c * c - 1.5};
                double ra = 0.0, rb = 0.0, cc = 0.0;
                for (int m = 0; m < M; ++m) {
                    double A = 0.0, B = 0.0;
                    for (int l = 0; l < L; ++l) {
                        A += Fd[K + m * L + l] * P[l];
                        B += Fd[K + m * L + l] * dP[l];
                    }
                    ra += df[m][a] * f[m][b] * A;
                    rb += f[m][a] * df[m][b] * A;
                    cc += f[m][a] * f[m][b] * B;
                }
                ra *= 2.0; rb *= 2.0; cc *= 2.0;
                // d cos / d r^ij = (u^ik - cos u^ij) / r_ij
                const double ca = cc * ir[a], cb = cc * ir[b];
                px[a] += ra * ux[a] + ca * (ux[b] - c * ux[a]);
                py[a] += ra * uy[a] + ca * (uy[b] - c * uy[a]);
                pz[a] += ra * uz[a] + ca * (uz[b] - c * uz[a]);
                px[b] += rb * ux[b] + cb * (ux[a] - c * ux[b]);
                py[b] += rb * uy[b] + cb * (uy[a] - c * uy[b]);
                pz[b] += rb * uz[b] + cb * (uz[a] - c * uz[b]);
            }
        for (int k = 0, a = 0; k < cnt; ++k) {
            const bool hit = a < n && ek[a] == k;
            part[(size_t)(k * 3 + 0) * d.Npad] = hit ? px[a] : 0.0;
            part[(size_t)(k * 3 + 1) * d.Npad] = hit ? py[a] : 0.0;
            part[(size_t)(k * 3 + 2) * d.Npad] = hit ? pz[a] : 0.0;
            if (hit) ++a;
        }
    }
    block_sum<1>(ui, red);
    if (threadIdx.x == 0) d.part_force[((size_t)slot * d.nblk_atom + blockIdx.x) * kNForcePart + 7] = ui[0];
}

void launch_force_dn(const Dev &d, int p_lo, cudaStream_t st) {
    const int nimg = images_in_grid(d.S, p_lo);
    if (nimg <= 0) return;
    dim3 grid(d.nblk_atom, nimg);
    dn_partial_kernel<<<grid, kThreadsAtom, 0, st>>>(d, p_lo);
    launch_pair_forces_manybody(d, p_lo, st);
}

}  // namespace cfn
